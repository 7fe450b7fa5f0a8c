// vc_line.cuh — step a7, the two-claims -> one-claim line restriction (reading c-5; absent from
// PAPER.md, which defers to [8],[10] at PAPER.md:85):
//   q[t] = V~_{i+1}(l(t)),  l(t) = r1 + t (r2 - r1),  t = 0..s  (q[0] = v1, q[1] = v2 come from the folds),
//   tau = draw;  z <- l(tau);  claim <- q(tau) by Lagrange interpolation on nodes 0..s.
// ONE pass over V_{i+1} serves all s-1 evaluation points: each thread keeps 2^nt consecutive words
// in registers, folds them with the first nt coordinates of l(t) (2^nt - 1 multiplies), and weights
// the result with eq(rest of its index, rest of l(t)) read from a per-block table built by doubling.
#pragma once
#include "vc_kernels.cuh"

namespace vc {

constexpr int LINE_NT = 3;   // variables folded inside a thread (8 words per thread)
constexpr int LINE_TB = 8;   // variables covered by the 256 threads of a block

// dynamic shared memory layout: pts[(s-1)*s] | W[(s-1)*256] | red[(s-1)*8] | qs[s+1]
__host__ __device__ inline size_t line_smem_words(uint32_t s) {
    const size_t m = s > 1 ? s - 1 : 0;
    return m * s + m * 256 + m * 8 + (s + 1) + 32;
}

static __global__ void __launch_bounds__(256)
k_line(const uint64_t *__restrict__ Vb, uint32_t s, DevState *st, uint64_t *part, uint64_t *tr_q) {
    extern __shared__ uint64_t sm[];
    __shared__ int s_last;
    const uint32_t m = s - 1;                      // number of evaluation points t = 2..s
    uint64_t *pts = sm;                            // pts[(t-2)*s + k] = l(t)_k
    uint64_t *Wt = pts + (size_t)m * s;            // Wt[(t-2)*256 + tid]
    uint64_t *red = Wt + (size_t)m * 256;          // red[(t-2)*8 + warp]
    uint64_t *qs = red + (size_t)m * 8;            // q[0..s]
    uint64_t *red1 = qs + (s + 1);                 // 32 words for block_sum<1>
    const uint32_t nt = s < LINE_NT ? s : LINE_NT;
    const uint32_t tb = (s - nt) < LINE_TB ? (s - nt) : LINE_TB;
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    if (m > 0) {
        for (uint32_t i = tid; i < m * s; i += blockDim.x) {
            const uint32_t t = i / s + 2, k = i % s;
            const uint64_t a = st->r1[k], b = st->r2[k];
            pts[i] = fp61::add(a, fp61::mul(t, fp61::sub(b, a)));
        }
        __syncthreads();
        // seed of each table: the block's fixed high bits
        for (uint32_t t = tid; t < m; t += blockDim.x) {
            uint64_t e = 1;
            for (uint32_t k = nt + tb; k < s; k++)
                e = fp61::mul(e, fp61::chi((blockIdx.x >> (k - nt - tb)) & 1u, pts[t * s + k]));
            Wt[t * 256] = e;
        }
        __syncthreads();
        for (uint32_t k = 0; k < tb; k++) {
            const uint32_t half = 1u << k;
            for (uint32_t i = tid; i < m * half; i += blockDim.x) {
                const uint32_t t = i >> k, u = i & (half - 1);
                const uint64_t e = Wt[t * 256 + u], hi = fp61::mul(e, pts[t * s + nt + k]);
                Wt[t * 256 + u + half] = hi;
                Wt[t * 256 + u] = fp61::sub(e, hi);
            }
            __syncthreads();
        }
        // one pass over V_{i+1}: 2^nt words per thread, kept in registers for all t
        const bool active = tid < (1u << tb);
        uint64_t v[1 << LINE_NT];
        const size_t base = (((size_t)blockIdx.x << tb) + tid) << nt;
#pragma unroll
        for (int e = 0; e < (1 << LINE_NT); e++) v[e] = (active && e < (1 << nt)) ? Vb[base + e] : 0;
        for (uint32_t t = 0; t < m; t++) {
            uint64_t f[1 << LINE_NT];
#pragma unroll
            for (int e = 0; e < (1 << LINE_NT); e++) f[e] = v[e];
#pragma unroll
            for (int k = 0; k < LINE_NT; k++) {
                if (k < (int)nt) {
                    const uint64_t x = pts[t * s + k];
#pragma unroll
                    for (int e = 0; e < ((1 << LINE_NT) >> (k + 1)); e++)
                        f[e] = fp61::add(f[2 * e], fp61::mul(x, fp61::sub(f[2 * e + 1], f[2 * e])));
                }
            }
            uint64_t val = active ? fp61::mul(f[0], Wt[t * 256 + tid]) : 0;
            val = warp_sum(val);
            if (lane == 0) red[t * 8 + warp] = val;
        }
        __syncthreads();
        for (uint32_t t = tid; t < m; t += blockDim.x) {
            uint64_t a = 0;
            for (uint32_t w = 0; w < (blockDim.x >> 5); w++) a = fp61::add(a, red[t * 8 + w]);
            __stcg(&part[(size_t)blockIdx.x * m + t], a);
        }
    }
    // last-block-done
    __threadfence();
    __syncthreads();
    if (tid == 0) {
        unsigned tk = atomicAdd(&st->ticket, 1u);
        s_last = (tk == gridDim.x - 1);
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    for (uint32_t t = warp; t < m; t += (blockDim.x >> 5)) {
        uint64_t a = 0;
        for (uint32_t b = lane; b < gridDim.x; b += 32) a = fp61::add(a, __ldcg(&part[(size_t)b * m + t]));
        a = warp_sum(a);
        if (lane == 0) qs[t + 2] = a;
    }
    if (tid == 0) { qs[0] = st->v1; qs[1] = st->v2; st->ticket = 0; }
    __syncthreads();
    const uint64_t tau = fp61::draw(st->seed, st->ctr);
    for (uint32_t k = tid; k <= s; k += blockDim.x) tr_q[k] = qs[k];
    // claim <- sum_k q[k] L_k(tau),  L_k(tau) = prod_{m != k}(tau - m) * (-1)^{s-k} / (k! (s-k)!)
    uint64_t term = 0;
    if (tid <= s) {
        uint64_t num = 1;
        for (uint32_t mm = 0; mm <= s; mm++)
            if (mm != tid) num = fp61::mul(num, fp61::sub(tau, mm));
        uint64_t dinv = fp61::mul(st->invfact[tid], st->invfact[s - tid]);
        term = fp61::mul(qs[tid], fp61::mul(num, dinv));
        if ((s - tid) & 1u) term = fp61::neg(term);
    }
    uint64_t tv[1] = {term};
    block_sum<1>(tv, red1);
    // z <- l(tau)   (reads r1,r2 before anyone overwrites them: same block, ordered by the barrier below)
    uint64_t znew = 0;
    if (tid < s) { const uint64_t a = st->r1[tid], b = st->r2[tid]; znew = fp61::add(a, fp61::mul(tau, fp61::sub(b, a))); }
    __syncthreads();
    if (tid < s) st->z[tid] = znew;
    if (tid == 0) { st->claim = tv[0]; st->ctr += 1; }
}

}  // namespace vc
