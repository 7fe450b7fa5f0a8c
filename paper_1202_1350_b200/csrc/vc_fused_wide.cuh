// vc_fused_wide.cuh — one layer on the whole grid (steps a3-a7), called from k_fused by every CTA.
#pragma once
#include "vc_fused.cuh"

namespace vc {

// Where a CTA keeps the per-gate state of its chunks.
//   RES = true : shared memory (<= F_MAXK chunks per CTA): sP weight, sW fixed operand, sI1 = in1 | type<<30, sI2 = in2
//   RES = false: global memory (layer wider than gridDim * F_MAXK chunks): weights in a.P, records re-read
struct GateState {
    uint64_t *sP, *sW;
    uint32_t *sI1, *sI2;
};

template <bool RES>
__device__ __forceinline__ void wide_layer(const FusedArgs &a, FusedCtx &cx, uint8_t *dyn, uint32_t layer, uint64_t *tr) {
    const uint32_t tid = threadIdx.x, G = gridDim.x, b = blockIdx.x;
    const LayerDesc Li = a.L[layer], Lb = a.L[layer + 1];
    const uint32_t si = Li.log_n, s = Lb.log_n;
    const uint32_t n = 1u << si;
    const uint64_t *__restrict__ Vb = Lb.V;
    const uint32_t nch = n >> F_CHUNK_LOG ? n >> F_CHUNK_LOG : 1;
    const uint32_t c0 = (uint32_t)(((uint64_t)b * nch) / G), c1 = (uint32_t)(((uint64_t)(b + 1) * nch) / G);
    const uint32_t nk = c1 - c0;
    GateState gs;
    gs.sP = reinterpret_cast<uint64_t *>(dyn);
    gs.sW = gs.sP + F_MAXK * FT;
    gs.sI1 = reinterpret_cast<uint32_t *>(gs.sW + F_MAXK * FT);
    gs.sI2 = gs.sI1 + F_MAXK * FT;
    uint64_t *Elo = gs.sW;                       // beta low table aliases sW until the records are loaded

    // ---- a3: P[g] = eq(g,z) = Elo[g & 1023] * Ehi[g >> 10]
    const uint32_t cl = si < F_CHUNK_LOG ? si : F_CHUNK_LOG;
    build_eq_low(Elo, cx.z, cl);
    const uint64_t elo = tid < (1u << cl) ? Elo[tid] : 0;
    uint64_t claim_part = 0;
    for (uint32_t k = 0; k < nk; k++) {
        const uint32_t c = c0 + k, g = (c << F_CHUNK_LOG) + tid;
        uint64_t e = elo;
        for (uint32_t kk = F_CHUNK_LOG; kk < si; kk++) e = fp61::mul(e, fp61::chi((c >> (kk - F_CHUNK_LOG)) & 1u, cx.z[kk]));
        if (RES) gs.sP[k * FT + tid] = e; else if (g < n) a.P[g] = e;
        if (layer == 0 && g < n) claim_part = fp61::add(claim_part, fp61::mul(e, Li.V[g]));
    }
    if (layer == 0) {                            // a2: start claim V~_0(z_0) = sum_g beta(z_0,g) V_0[g]
        uint64_t v[3] = {claim_part, 0, 0};
        block_reduce3(cx, v);
        grid_allreduce(cx, a, 1);
        if (tid == 0) cx.claim = cx.acc[0];
    }
    __syncthreads();                             // Elo (aliasing sW) is dead from here
    if (RES) {
        for (uint32_t k = 0; k < nk; k++) {
            const uint32_t g = ((c0 + k) << F_CHUNK_LOG) + tid;
            uint32_t i1 = 0, i2 = 0, t = 3;
            uint64_t w = 0;
            if (g < n) { i1 = Li.in1[g]; i2 = Li.in2[g]; t = Li.type[g]; w = Vb[i2]; }
            else gs.sP[k * FT + tid] = 0;        // padding gates of a short layer carry weight 0
            gs.sI1[k * FT + tid] = i1 | (t << 30);
            gs.sI2[k * FT + tid] = i2;
            gs.sW[k * FT + tid] = w;
        }
    }

    // ---- a4-a6: 2s rounds
    uint64_t r_prev = 0;
    uint32_t upd_bit = 0;
    bool have_upd = false, upd_in1 = true;
    for (int phase = 1; phase <= 2; phase++) {
        for (uint32_t j = 0; j < s; j++) {
            const uint64_t omr = fp61::sub(1, r_prev);
            // table of the previous round (materialised): j=0 none needed, j=1: V_{i+1}, j>=2: T[(j-2)&1]
            const uint64_t *Aprev = j <= 1 ? Vb : ((j & 1) ? a.T1 : a.T0);   // A_{j-1}
            uint64_t *Aout = (j & 1) ? a.T0 : a.T1;                            // A_j (for j >= 1)
            acc128 a0, a1, a2; a0.clear(); a1.clear(); a2.clear();
            const uint64_t v1 = cx.v1;
            for (uint32_t k = 0; k < nk; k++) {
                const uint32_t g = ((c0 + k) << F_CHUNK_LOG) + tid;
                uint32_t i1, i2, t; uint64_t Pg, w = 0;
                if (RES) {
                    i1 = gs.sI1[k * FT + tid]; i2 = gs.sI2[k * FT + tid]; Pg = gs.sP[k * FT + tid];
                    t = i1 >> 30; i1 &= 0x3fffffffu;
                    if (phase == 1) w = gs.sW[k * FT + tid];
                } else {
                    if (g >= n) continue;
                    i1 = Li.in1[g]; i2 = Li.in2[g]; t = Li.type[g]; Pg = a.P[g];
                    if (phase == 1) w = Vb[i2];
                }
                if (have_upd) {
                    const uint32_t ub = ((upd_in1 ? i1 : i2) >> upd_bit) & 1u;
                    Pg = fp61::mul(Pg, ub ? r_prev : omr);
                    if (RES) gs.sP[k * FT + tid] = Pg; else a.P[g] = Pg;
                }
                const uint32_t idx = phase == 1 ? i1 : i2;
                const uint32_t bit = (idx >> j) & 1u, u = idx >> (j + 1);
                uint64_t lo, hi;
                if (j == 0) {
                    const ulonglong2 pr = *reinterpret_cast<const ulonglong2 *>(Vb + 2 * (size_t)u);
                    lo = pr.x; hi = pr.y;
                } else {                         // fold A_{j-1} on the fly with r_{j-1}: no second rendezvous
                    const ulonglong2 p0 = __ldcg(reinterpret_cast<const ulonglong2 *>(Aprev + 4 * (size_t)u));
                    const ulonglong2 p1 = __ldcg(reinterpret_cast<const ulonglong2 *>(Aprev + 4 * (size_t)u + 2));
                    lo = fold2(p0.x, p0.y, r_prev); hi = fold2(p1.x, p1.y, r_prev);
                }
                if (phase == 1) gate_terms<1>(t, Pg, w, bit, lo, hi, a0, a1, a2);
                else gate_terms<2>(t, Pg, v1, bit, lo, hi, a0, a1, a2);
            }
            // materialise A_j for the next round's on-the-fly fold (2^(s-j) words, spread over the grid)
            if (j >= 1) {
                const uint32_t cnt = 1u << (s - j);
                for (uint32_t v = b * FT + tid; v < cnt; v += G * FT) {
                    const ulonglong2 pr = __ldcg(reinterpret_cast<const ulonglong2 *>(Aprev + 2 * (size_t)v));
                    __stcg(Aout + v, fold2(pr.x, pr.y, r_prev));
                }
            }
            uint64_t v3[3] = {a0.value(), a1.value(), a2.value()};
            block_reduce3(cx, v3);
            grid_allreduce(cx, a, 3);
            const uint64_t r = fp61::draw(cx.seed, cx.ctr);
            if (b == 0 && tid < 3) tr[tid] = cx.acc[tid];
            tr += 3;
            __syncthreads();
            if (tid == 0) { cx.ctr += 1; if (phase == 1) cx.r1[j] = r; else cx.r2[j] = r; }
            // pending weight update for the next round
            have_upd = true; upd_in1 = (phase == 1); upd_bit = j; r_prev = r;
        }
        // V~_{i+1}(r) = fold of the last materialised table (2 words) with the last challenge
        if (tid == 0) {
            const uint64_t *Alast = s == 1 ? Vb : (((s - 1) & 1) ? a.T0 : a.T1);
            const uint64_t x0 = __ldcg(Alast), x1 = __ldcg(Alast + 1);
            const uint64_t val = fold2(x0, x1, r_prev);
            if (phase == 1) cx.v1 = val; else cx.v2 = val;
        }
        __syncthreads();
    }
    // ---- a7: line restriction, all CTAs share the pass over V_{i+1}
    if (s > 1) {
        line_partials(Vb, s, cx, reinterpret_cast<uint64_t *>(dyn), b, G);
        grid_allreduce(cx, a, s - 1);
    }
    line_finish(s, cx, a.st, tr, b == 0);
}

}  // namespace vc
