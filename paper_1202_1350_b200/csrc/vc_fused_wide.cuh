// vc_fused_wide.cuh — one layer on the whole grid (steps a2-a7), called from k_fused by every CTA.
//
// Gate state per gate: W (weight with the fixed operand folded in for MULT), c (additive constant), idx (the index
// being bound in this phase; bit 31 = "x ignored").  RES = true keeps it in shared memory, RES = false in global
// scratch (layers with more than `cap` gates per CTA).
// Fold tables, per phase (mode from the load-time plan):
//   F_MODE_SLICE : level 0 is V_{i+1} in L2; levels 1..K-1 are the slice this CTA's gates read, folded locally in
//                  shared memory; level K-1 of the WHOLE table is published once (each CTA computes the entries it
//                  owns straight from V_{i+1} with an eq table of the first K-1 challenges) and from level K on every
//                  CTA folds the whole (<= 2^10-entry) table itself.  No table traffic through L2 after that.
//   F_MODE_GLOBAL: every level is materialised in global memory by the whole grid and the gates fold level j-1 on the
//                  fly (two extra multiplies per gate-round); used when a CTA's slice would not fit.
#pragma once
#include "vc_fused.cuh"
#include "vc_fused_line.cuh"
#include "vc_fused_small.cuh"

namespace vc {

// level K-1 of the fold table, entries [e0, e1): T[e] = sum_v eq(v, rr[0..K-1)) V[e 2^(K-1) + v].  One warp per entry.
__device__ __forceinline__ void publish_level(const uint64_t *__restrict__ Vb, const uint64_t *rr, uint32_t km1, uint32_t e0,
                                              uint32_t e1, uint64_t *eqt, uint64_t *Tg) {
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    __syncthreads();                                             // rr[km1-1] (written by the last rendezvous) is visible
    for (uint32_t v = tid; v < (1u << km1); v += FT) eqt[v] = eq_direct(v, rr, 0, km1);
    __syncthreads();
    for (uint32_t e = e0 + warp; e < e1; e += FT / 32) {
        const uint64_t *src = Vb + ((size_t)e << km1);
        acc128 A; A.clear();
        uint64_t sum = 0; uint32_t it = 0;
        for (uint32_t v = lane; v < (1u << km1); v += 32) {
            A.mac(eqt[v], src[v]);
            if (++it == 32) { sum = fp61::add(sum, A.value()); A.clear(); it = 0; }
        }
        sum = warp_sum61(fp61::add(sum, A.value()));
        if (lane == 0) __stcg(Tg + e, sum);
    }
}

template <bool RES>
__device__ __forceinline__ void wide_layer(const FusedArgs &a, FusedCtx &cx, const uint64_t *invfact, uint8_t *dyn,
                                           uint32_t layer, uint64_t *tr) {
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, G = gridDim.x, b = blockIdx.x;
    const LayerPlan &Lp = a.L[layer];
    const uint32_t si = Lp.log_n, s = a.L[layer + 1].log_n;
    const uint64_t *__restrict__ Vb = a.L[layer + 1].V;
    const uint8_t *__restrict__ gtype = Lp.type;
    const uint32_t *__restrict__ gin1 = Lp.in1, *__restrict__ gin2 = Lp.in2;
    const CtaPlan cp = Lp.cta[b];
    const uint32_t g0 = cp.g0, ng = cp.g1 - cp.g0;
    const uint32_t nk = (ng + FT - 1) / FT;
    const uint32_t nw = ng >= (uint32_t)FT ? (uint32_t)FT / 32 : (ng + 31) / 32;   // warps that own gates
    const uint32_t cap = Lp.cap;
    uint64_t *sW = reinterpret_cast<uint64_t *>(dyn);
    uint64_t *sC = sW + cap;
    uint32_t *sI = reinterpret_cast<uint32_t *>(sC + cap);
    uint64_t *bufX = reinterpret_cast<uint64_t *>(dyn + Lp.off_tab), *bufY = bufX + Lp.xw;
    uint64_t *scr = reinterpret_cast<uint64_t *>(dyn + Lp.off_scr);
    const uint64_t seed = cx.seed;

    // ---- a3: beta(z, g) through a two-level eq table (built in the fold buffers, which are idle until level 1)
    __syncthreads();
    uint32_t ctr = (uint32_t)cx.ctr;
    const EqTab eb = build_eq_tab(bufX, bufX + (1u << F_EQLOG), cx.z, si, tid, FT);
    __syncthreads();
    uint64_t claim_part = 0;
    for (uint32_t k = 0; k < nk; k++) {
        const uint32_t l = k * FT + tid;
        if (l >= ng) break;
        const uint32_t g = g0 + l;
        const uint64_t P = eb.eq_of(g);
        const uint32_t i1 = gin1[g], i2 = gin2[g], t = gtype[g];
        uint64_t W, c; uint32_t ign;
        gate_state(1, t, P, Vb[i2], W, c, ign);
        if (RES) { sW[l] = W; sC[l] = c; sI[l] = i1; } else { a.P[g] = W; a.C[g] = c; }
        if (layer == 0) claim_part = fp61::add(claim_part, fp61::mul(P, Lp.V[g]));
    }
    if (layer == 0) {                            // a2: start claim V~_0(z_0) = sum_g beta(z_0,g) V_0[g]
        claim_part = warp_sum61(claim_part);
        if (lane == 0) cx.red[warp * 4] = claim_part;
        __syncthreads();
        if (warp == 0) { const uint64_t t0 = warp_sum61(lane < (uint32_t)FT / 32 ? cx.red[lane * 4] : 0); if (lane == 0) cx.acc[0] = t0; }
        grid_allreduce(cx, a, 1, false);
        if (tid == 0) cx.claim = cx.acc[0];
    }

    VC_TR(11);
    for (int ph = 0; ph < 2; ph++) {
        const uint32_t mode = Lp.mode[ph], K = Lp.K[ph], blo = cp.blo[ph], nbk = cp.nb[ph];
        uint64_t *rr = ph == 0 ? cx.r1 : cx.r2;
        if (ph == 1) {
            // ---- phase switch: plain weight P = beta(z,g) eq(in1[g], r1), then the phase-2 state
            __syncthreads();                     // v1, r1[s-1] visible; phase-1 tables dead
            const uint64_t v1 = cx.v1;
            const EqTab e0 = build_eq_tab(bufX, bufX + (1u << F_EQLOG), cx.z, si, tid, FT);
            const EqTab e1 = build_eq_tab(bufX + (2u << F_EQLOG), bufX + (3u << F_EQLOG), cx.r1, s, tid, FT);
            __syncthreads();
            for (uint32_t k = 0; k < nk; k++) {
                const uint32_t l = k * FT + tid;
                if (l >= ng) break;
                const uint32_t g = g0 + l;
                const uint32_t i1 = gin1[g], i2 = gin2[g], t = gtype[g];
                const uint64_t P = fp61::mul(e0.eq_of(g), e1.eq_of(i1));
                uint64_t W, c; uint32_t ign;
                gate_state(2, t, P, v1, W, c, ign);
                if (RES) { sW[l] = W; sC[l] = c; sI[l] = i2 | (ign << 31); } else { a.P[g] = W; a.C[g] = c; }
            }
            __syncthreads();                     // tables free again before level 1 of phase 2 is built
        }
        uint64_t r_prev = 0;
        VC_TR(12);
        for (uint32_t j = 0; j < s; j++) {
            bool fence = false;
            const uint64_t *tab = Vb;            // level j as the gates see it (SLICE), or level j-1 (GLOBAL)
            uint32_t base = 0;
            if (mode == F_MODE_SLICE) {
                if (j >= 1) {
                    uint64_t *dst = (j & 1) ? bufX : bufY;
                    const uint64_t *prev = (j & 1) ? bufY : bufX;
                    if (j < K) {                 // this CTA's slice: nbk blocks of 2^(K-j) entries
                        const uint32_t cnt = nbk << (K - j);
                        if (j == 1) {
                            const uint64_t *src = Vb + ((size_t)blo << K);
                            for (uint32_t v = tid; v < cnt; v += FT) {
                                const ulonglong2 p = *reinterpret_cast<const ulonglong2 *>(src + 2 * (size_t)v);
                                dst[v] = fold2(p.x, p.y, r_prev);
                            }
                        } else {
                            for (uint32_t v = tid; v < cnt; v += FT) dst[v] = fold2(prev[2 * v], prev[2 * v + 1], r_prev);
                        }
                        base = blo << (K - j);
                    } else {                     // the whole table: from the published level K-1 (j = K >= 2), from V (j = 1),
                        const uint32_t cnt = 1u << (s - j);                         // else from the previous buffer
                        if (j == 1 || j == K) {
                            const uint64_t *src = j == 1 ? Vb : a.Tg;
                            for (uint32_t v = tid; v < cnt; v += FT) {
                                const ulonglong2 p = __ldcg(reinterpret_cast<const ulonglong2 *>(src + 2 * (size_t)v));
                                dst[v] = fold2(p.x, p.y, r_prev);
                            }
                        } else {
                            for (uint32_t v = tid; v < cnt; v += FT) dst[v] = fold2(prev[2 * v], prev[2 * v + 1], r_prev);
                        }
                    }
                    tab = dst;
                }
                if (K >= 2 && j == K - 1) {      // publish level K-1 for the next round (needs r_0..r_{K-2})
                    const uint32_t E = 1u << (s - K + 1);
                    publish_level(Vb, rr, K - 1, (uint32_t)(((uint64_t)b * E) / G), (uint32_t)(((uint64_t)(b + 1) * E) / G), scr, a.Tg);
                    fence = true;
                }
            } else {                             // GLOBAL: materialise level j (j >= 1) for the next round's on-the-fly fold
                tab = j <= 1 ? Vb : ((j & 1) ? a.T1 : a.T0);                       // level j-1
                if (j >= 1) {
                    uint64_t *Aout = (j & 1) ? a.T0 : a.T1;                          // level j
                    const uint32_t cnt = 1u << (s - j);
                    for (uint32_t v = b * FT + tid; v < cnt; v += G * FT) {
                        const ulonglong2 p = __ldcg(reinterpret_cast<const ulonglong2 *>(tab + 2 * (size_t)v));
                        __stcg(Aout + v, fold2(p.x, p.y, r_prev));
                    }
                }
                fence = true;
            }
            VC_TR(13);
            __syncthreads();                     // level j ready in shared memory
            VC_TR(14);
            // ---- a4 (+ the pending a6 weight update): every gate of this CTA
            if (warp < nw) {
                const uint64_t omr = fp61::sub(1, r_prev);
                acc128 X, X1, Y, Y1; X.clear(); X1.clear(); Y.clear(); Y1.clear();
                uint64_t gs[3] = {0, 0, 0};
                for (uint32_t k = 0; k < nk; k++) {
                    const uint32_t l = k * FT + tid;
                    if (l >= ng) break;
                    uint64_t W, c; uint32_t idx;
                    if (RES) { W = sW[l]; c = sC[l]; idx = sI[l]; }
                    else {
                        const uint32_t g = g0 + l;
                        W = a.P[g]; c = a.C[g];
                        idx = ph == 0 ? gin1[g] : (gin2[g] | ((gtype[g] == VC_RELAY ? 1u : 0u) << 31));
                    }
                    if (j >= 1) {
                        W = fp61::mul(W, ((idx >> (j - 1)) & 1u) ? r_prev : omr);
                        if (RES) sW[l] = W; else a.P[g0 + l] = W;
                    }
                    const uint32_t bit = (idx >> j) & 1u, u = (idx & F_IDX_MASK) >> (j + 1);
                    uint64_t lo, hi;
                    if (mode == F_MODE_SLICE || j == 0) {
                        const ulonglong2 p = *reinterpret_cast<const ulonglong2 *>(tab + (2 * (size_t)u - base));
                        lo = p.x; hi = p.y;
                    } else {                     // fold level j-1 on the fly with r_{j-1}
                        const ulonglong2 p0 = __ldcg(reinterpret_cast<const ulonglong2 *>(tab + 4 * (size_t)u));
                        const ulonglong2 p1 = __ldcg(reinterpret_cast<const ulonglong2 *>(tab + 4 * (size_t)u + 2));
                        lo = fold2(p0.x, p0.y, r_prev); hi = fold2(p1.x, p1.y, r_prev);
                    }
                    if (idx >> 31) { lo = 0; hi = 0; }
                    gate_mac(W, c, bit, lo, hi, X, X1, Y, Y1);
                    if ((k & 7) == 7) {          // 8 products per accumulator at most
                        uint64_t g3[3];
                        gate_fin(X, X1, Y, Y1, g3);
#pragma unroll
                        for (int q = 0; q < 3; q++) gs[q] = fp61::add(gs[q], g3[q]);
                        X.clear(); X1.clear(); Y.clear(); Y1.clear();
                    }
                }
                uint64_t g3[3];
                gate_fin(X, X1, Y, Y1, g3);
#pragma unroll
                for (int q = 0; q < 3; q++) {
                    const uint64_t v = warp_sum61(fp61::add(gs[q], g3[q]));
                    if (lane == 0) cx.red[warp * 4 + q] = v;
                }
            }
            // ---- a5 + a6: grid reduction of the three round values, then the challenge
            uint64_t *rslot = rr + j;
            VC_TR(15);
            round_allreduce(cx, a, nw, fence, tr, rslot, seed, ctr);
            VC_TR(16);
            ctr++;
            tr += 3;
            r_prev = *rslot;
        }
        // ---- V~_{i+1}(r) = the two entries of level s-1 folded with the last challenge
        if (tid == 0) {
            uint64_t x0, x1;
            if (mode == F_MODE_SLICE) {
                const uint64_t *t1 = s == 1 ? Vb : (((s - 1) & 1) ? bufX : bufY);
                x0 = t1[0]; x1 = t1[1];
            } else {
                const uint64_t *t1 = s == 1 ? Vb : (((s - 1) & 1) ? a.T0 : a.T1);
                x0 = __ldcg(t1); x1 = __ldcg(t1 + 1);
            }
            const uint64_t val = fold2(x0, x1, r_prev);
            if (ph == 0) cx.v1 = val; else cx.v2 = val;
        }
    }
    if (tid == 0) cx.ctr = ctr;
    if (b == 0 && warp == 2) transcript_flush(cx, a);       // the last round's message
    __syncthreads();
    VC_TR(17);
    // ---- a7: line restriction, all CTAs share the pass over V_{i+1}
    if (s > 1) {
        line_partials(Vb, s, cx, bufX, b, G, tid, FT);
        grid_allreduce(cx, a, s - 1, false);
    }
    VC_TR(18);
    line_finish(s, cx, invfact, tr, b == 0, tid);
    __syncthreads();
    VC_TR(19);
}

}  // namespace vc
