// vc_kernels.cuh — "streaming" schedule: one kernel launch per protocol step, every buffer in HBM/L2.
// Steps a1-a7 of SURVEY.md §8(a).  Used for layers too wide for the on-chip schedule and as the
// always-available baseline schedule (vc_set_schedule(c, 1)).
//
// Method (§4.1.1): each gate contributes independently to each message; one pass
// over the layer's gates per message; contributions reduced in F_p.  The paper's temporary array +
// Thrust reduction is replaced by 128-bit lazy register accumulators,
// warp shuffles, one 3-word partial per block and a last-block-done finalisation that also draws
// the next challenge on the device (north_star (3)).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "fp61.cuh"
#include "vc_state.cuh"

namespace vc {

using fp61::acc128;

__device__ __forceinline__ uint64_t shfl_down64(uint64_t v, int d) {
    return __shfl_down_sync(0xffffffffu, v, d);
}
__device__ __forceinline__ uint64_t warp_sum(uint64_t v) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v = fp61::add(v, shfl_down64(v, d));
    return v;  // valid on lane 0
}

// Block-wide sum mod p of K words per thread; result valid on thread 0.  red: K*32 words of smem.
template <int K>
__device__ __forceinline__ void block_sum(uint64_t (&v)[K], uint64_t *red) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
#pragma unroll
    for (int k = 0; k < K; k++) v[k] = warp_sum(v[k]);
    __syncthreads();  // red may still be in use by a previous call
    if (lane == 0) {
#pragma unroll
        for (int k = 0; k < K; k++) red[k * 32 + warp] = v[k];
    }
    __syncthreads();
    if (warp == 0) {
#pragma unroll
        for (int k = 0; k < K; k++) {
            uint64_t x = lane < nw ? red[k * 32 + lane] : 0;
            v[k] = warp_sum(x);
        }
    }
}

// Grid-wide sum mod p: every block publishes K words; the block that takes the last ticket sums all
// partials.  Returns true in every thread of that last block; totals valid on its thread 0.
template <int K>
__device__ __forceinline__ bool grid_sum_last_block(uint64_t (&v)[K], uint64_t *part, DevState *st, uint64_t *red) {
    __shared__ int s_last;
    block_sum<K>(v, red);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int k = 0; k < K; k++) __stcg(&part[(size_t)blockIdx.x * K + k], v[k]);
        __threadfence();
        unsigned t = atomicAdd(&st->ticket, 1u);
        s_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!s_last) return false;
    __threadfence();
#pragma unroll
    for (int k = 0; k < K; k++) {
        uint64_t a = 0;
        for (unsigned b = threadIdx.x; b < gridDim.x; b += blockDim.x) a = fp61::add(a, __ldcg(&part[(size_t)b * K + k]));
        v[k] = a;
    }
    block_sum<K>(v, red);
    if (threadIdx.x == 0) st->ticket = 0;
    return true;
}

// ------------------------------------------------------------------ a1: evaluation
// V_d <- input (checked canonical)
static __global__ void k_copy_input(const uint64_t *in, uint64_t *out, uint64_t n, DevState *st) {  // in may equal out
    unsigned bad = 0;
    for (uint64_t i = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x) {
        uint64_t w = in[i];
        bad |= (w >= fp61::P);
        out[i] = w;
    }
    if (bad) atomicOr(&st->flags, 1u);
}

__device__ __forceinline__ uint64_t gate_f(uint32_t t, uint64_t L, uint64_t R) {
    // VC_ADD L+R, VC_MULT L*R, VC_SUB L-R, VC_RELAY L   (reading c-3)
    uint64_t r = L;
    if (t == 0) r = fp61::add(L, R);
    else if (t == 1) r = fp61::mul(L, R);
    else if (t == 2) r = fp61::sub(L, R);
    return r;
}

// V_i[g] = f_type(V_{i+1}[in1[g]], V_{i+1}[in2[g]])   (all gates of a layer in parallel)
static __global__ void k_eval(const uint8_t *__restrict__ type, const uint32_t *__restrict__ in1,
                       const uint32_t *__restrict__ in2, const uint64_t *__restrict__ Vb,
                       uint64_t *__restrict__ Vout, uint64_t *__restrict__ Vout2, uint32_t n) {
    for (uint32_t g = blockIdx.x * blockDim.x + threadIdx.x; g < n; g += gridDim.x * blockDim.x) {
        uint64_t v = gate_f(type[g], Vb[in1[g]], Vb[in2[g]]);
        Vout[g] = v;
        if (Vout2) Vout2[g] = v;
    }
}

// ------------------------------------------------------------------ a2: start of the proof
// ctr <- 0; z_0 <- s0 draws.  One warp-sized block.
static __global__ void k_start(DevState *st, uint64_t seed, uint32_t s0) {
    for (uint32_t k = threadIdx.x; k < s0; k += blockDim.x) st->z[k] = fp61::draw(seed, k);
    if (threadIdx.x == 0) { st->seed = seed; st->ctr = s0; st->ticket = 0; }
}

// ------------------------------------------------------------------ a3: beta weights
// P[g] = eq(g,z) for g < 2^s.  Each block builds its 2^c-entry chunk by doubling in shared memory:
// T[u + 2^k] = T[u] z_k ; T[u] -= T[u + 2^k]   (1 multiply per new entry), seeded with the product
// over the bits >= c that are fixed for the chunk.
constexpr int BETA_LOG_CHUNK = 11;
static __global__ void __launch_bounds__(256) k_beta(const DevState *__restrict__ st, uint64_t *__restrict__ Pw, uint32_t s) {
    __shared__ uint64_t T[1 << BETA_LOG_CHUNK];
    const uint32_t c = s < BETA_LOG_CHUNK ? s : BETA_LOG_CHUNK;
    const uint32_t base = blockIdx.x << c;
    if (threadIdx.x == 0) {
        uint64_t e = 1;
        for (uint32_t k = c; k < s; k++) e = fp61::mul(e, fp61::chi((base >> k) & 1, st->z[k]));
        T[0] = e;
    }
    __syncthreads();
    for (uint32_t k = 0; k < c; k++) {
        const uint32_t half = 1u << k;
        const uint64_t zk = st->z[k];
        for (uint32_t u = threadIdx.x; u < half; u += blockDim.x) {
            uint64_t e = T[u], hi = fp61::mul(e, zk);
            T[u + half] = hi;
            T[u] = fp61::sub(e, hi);
        }
        __syncthreads();
    }
    for (uint32_t u = threadIdx.x; u < (1u << c); u += blockDim.x) Pw[base + u] = T[u];
}

// claim <- sum_g P[g] V_0[g] = V~_0(z_0)
static __global__ void __launch_bounds__(RED_BLOCK) k_dot_claim(const uint64_t *__restrict__ Pw, const uint64_t *__restrict__ V,
                                                          uint32_t n, uint64_t *part, DevState *st) {
    __shared__ uint64_t red[32];
    acc128 a; a.clear();
    uint64_t sum = 0; int it = 0;
    for (uint32_t g = blockIdx.x * blockDim.x + threadIdx.x; g < n; g += gridDim.x * blockDim.x) {
        a.mac(Pw[g], V[g]);
        if (++it == 32) { sum = fp61::add(sum, a.value()); a.clear(); it = 0; }
    }
    uint64_t v[1] = {fp61::add(sum, a.value())};
    if (grid_sum_last_block<1>(v, part, st, red) && threadIdx.x == 0) st->claim = v[0];
}

}  // namespace vc
