// vc_sum.cuh — the single sum gate of very large fan-in at the output (
// DESIGN.md reading c-19; the ABI side is VC_SUM in include/vc.h).
//
// y = sum_w V_1[w] = sum over the Boolean cube of the multilinear V~_1, so the layer's iteration is a sum-check over the
// s variables of V~_1 itself, bit 0 first.  Round j: (G0, G1) = sums of the even- and odd-indexed entries of the table
// folded by r_0..r_{j-1}; the challenge r_j is drawn on the device after both sums are complete; the table is folded by
// r_j; after s rounds the one remaining entry is the claim V~_1(r) and z' = r.
//
// Kernels (HBM-bound, 8 B per table word read once per round, half of it written):
//   k_sum_eval   V_0[0] = sum of V_1                                  (a1)
//   k_sum_first  G_0 from V_1, then r_0                               (last block done: message, draw)
//   k_sum_fold   T_{j+1} = fold(T_j, r_j) and, in the same pass, the two sums of T_{j+1} = message j+1, then r_{j+1}
//   k_sum_tail   one CTA: every remaining round once the table has at most 2^SUM_TAIL_LOG words
// The fold of round j and the sums of round j+1 share one pass over the table, so a round costs one read of T_j.
#pragma once
#include "vc_kernels.cuh"

namespace vc {

constexpr uint32_t SUM_TAIL_LOG = 11;     // 16 KB + 8 KB of static shared memory
constexpr int SUM_TAIL_T = 1024;

// the last block of a round: message out, next challenge in (the draw happens only here, after every partial is in)
__device__ __forceinline__ void sum_publish(DevState *st, uint64_t *tr, uint32_t j, uint64_t g0, uint64_t g1) {
    tr[2 * j] = g0; tr[2 * j + 1] = g1;
    const uint64_t r = fp61::draw(st->seed, st->ctr);
    st->ctr += 1;
    st->r = r;
    st->z[j] = r;
    st->G[0] = g0; st->G[1] = g1;
}

static __global__ void __launch_bounds__(RED_BLOCK) k_sum_eval(const uint64_t *__restrict__ Vb, uint64_t n, uint64_t *V0, uint64_t *out0,
                                                               uint64_t *part, DevState *st) {
    __shared__ uint64_t red[32];
    acc128 a; a.clear();
    for (uint64_t u = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; u < n; u += (uint64_t)gridDim.x * blockDim.x) a.addw(__ldcg(Vb + u));
    uint64_t v[1] = {a.value()};
    if (grid_sum_last_block<1>(v, part, st, red) && threadIdx.x == 0) { V0[0] = v[0]; if (out0) out0[0] = v[0]; }
}

// round 0: the sums of the even and odd entries of V_1 (n = 2^s words); starts the proof state of a sum-gate circuit
static __global__ void __launch_bounds__(RED_BLOCK) k_sum_first(const uint64_t *__restrict__ Vb, uint64_t n, uint64_t seed, uint64_t *part,
                                                                DevState *st, uint64_t *tr) {
    __shared__ uint64_t red[64];
    acc128 a0, a1; a0.clear(); a1.clear();
    const ulonglong2 *V2 = reinterpret_cast<const ulonglong2 *>(Vb);
    for (uint64_t u = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; u < n / 2; u += (uint64_t)gridDim.x * blockDim.x) {
        const ulonglong2 p = __ldcg(V2 + u);
        a0.addw(p.x); a1.addw(p.y);
    }
    uint64_t v[2] = {a0.value(), a1.value()};
    if (grid_sum_last_block<2>(v, part, st, red) && threadIdx.x == 0) {
        st->seed = seed; st->ctr = 0;                     // s_0 = 0: no draws for z_0; the start claim is V_0[0] itself
        sum_publish(st, tr, 0, v[0], v[1]);
    }
}

// round j -> j+1: Tout[u] = Tin[2u] + r_j (Tin[2u+1] - Tin[2u]) for u < half (= 2^(s-j-1)); message j+1 = the sums of the
// even / odd entries of Tout.  A thread folds two adjacent outputs, so its first goes to G0 and its second to G1.
// half == 1: Tout[0] is the final claim V~_1(r) and there is no further message.
static __global__ void __launch_bounds__(RED_BLOCK) k_sum_fold(const uint64_t *__restrict__ Tin, uint64_t *__restrict__ Tout, uint64_t half,
                                                               uint32_t j, uint64_t *part, DevState *st, uint64_t *tr) {
    __shared__ uint64_t red[64];
    const uint64_t r = st->r;
    if (half == 1) {
        if (blockIdx.x == 0 && threadIdx.x == 0) {
            const uint64_t lo = Tin[0], hi = Tin[1];
            const uint64_t c = fp61::add(lo, fp61::mul(r, fp61::sub(hi, lo)));
            Tout[0] = c; st->claim = c;
        }
        return;
    }
    acc128 a0, a1; a0.clear(); a1.clear();
    const ulonglong4 *T4 = reinterpret_cast<const ulonglong4 *>(Tin);
    ulonglong2 *O2 = reinterpret_cast<ulonglong2 *>(Tout);
    for (uint64_t u = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; u < half / 2; u += (uint64_t)gridDim.x * blockDim.x) {
        const ulonglong2 pa = __ldcg(reinterpret_cast<const ulonglong2 *>(T4 + u)), pb = __ldcg(reinterpret_cast<const ulonglong2 *>(T4 + u) + 1);
        ulonglong2 o;
        o.x = fp61::add(pa.x, fp61::mul(r, fp61::sub(pa.y, pa.x)));
        o.y = fp61::add(pb.x, fp61::mul(r, fp61::sub(pb.y, pb.x)));
        __stcg(O2 + u, o);
        a0.addw(o.x); a1.addw(o.y);
    }
    uint64_t v[2] = {a0.value(), a1.value()};
    if (grid_sum_last_block<2>(v, part, st, red) && threadIdx.x == 0) sum_publish(st, tr, j + 1, v[0], v[1]);
}

// one CTA finishes: T (2^m words, m <= SUM_TAIL_LOG) has had its sums published as message j0 and r_{j0} drawn; folds and
// sums ping-pong in shared memory for rounds j0+1 .. s-1, then the claim.
static __global__ void __launch_bounds__(SUM_TAIL_T) k_sum_tail(const uint64_t *__restrict__ Tin, uint32_t m, uint32_t j0, DevState *st, uint64_t *tr) {
    __shared__ uint64_t A[1u << SUM_TAIL_LOG], B[1u << (SUM_TAIL_LOG - 1)], red[64];
    __shared__ uint64_t s_r;
    const uint32_t tid = threadIdx.x;
    for (uint32_t u = tid; u < (1u << m); u += SUM_TAIL_T) A[u] = __ldcg(Tin + u);
    if (tid == 0) s_r = st->r;
    __syncthreads();
    uint64_t *cur = A, *nxt = B;
    for (uint32_t k = 0; k < m; k++) {                // fold by r_{j0+k}; then message j0+k+1 unless it was the last
        const uint32_t half = 1u << (m - k - 1);
        const uint64_t r = s_r;
        acc128 a0, a1; a0.clear(); a1.clear();
        for (uint32_t u = tid; u < half; u += SUM_TAIL_T) {
            const uint64_t lo = cur[2 * u], hi = cur[2 * u + 1];
            const uint64_t o = fp61::add(lo, fp61::mul(r, fp61::sub(hi, lo)));
            nxt[u] = o;
            if (u & 1) a1.addw(o); else a0.addw(o);
        }
        if (half == 1) {
            __syncthreads();
            if (tid == 0) st->claim = nxt[0];
            return;
        }
        uint64_t v[2] = {a0.value(), a1.value()};
        block_sum<2>(v, red);
        if (tid == 0) { sum_publish(st, tr, j0 + k + 1, v[0], v[1]); s_r = st->r; }
        __syncthreads();
        uint64_t *t = cur; cur = nxt; nxt = t;          // B holds 2^(m-1) words, then A's first quarter, and so on
    }
}

}  // namespace vc
