// vc_fused_thin.cuh — one grid-wide layer with at most one gate per worker thread (<= 480 gates per CTA): the
// latency-bound regime (steps a2-a7).  Same arithmetic as vc_fused_wide.cuh; what differs is the shape of a round:
//   * the gate (W, c, idx) lives in registers for the whole phase;
//   * warp specialisation: warps 0..14 are workers, warp 15 is the reducer.  A worker commits its two products of the
//     round (folded to one word each) to shared memory; after the commit barrier warp 0 posts the CTA's count to the
//     rendezvous word and waits, while the reducer sums the committed products into G[0..2] mod p and adds them to the
//     round's six data words, off the workers' critical path (software pipelining of step a5: the reduction of round j
//     overlaps round j+1; every contribution of message j is committed before challenge j is drawn);
//   * fold tables run one level behind: a gate folds the quad of level j-1 it needs itself (two extra multiplies on a
//     thread that has nothing else to do), and the workers build level j in the shadow of the rendezvous wait.
#pragma once
#include "vc_fused.cuh"
#include "vc_fused_line.cuh"
#include "vc_fused_small.cuh"
#include "vc_fused_wide.cuh"

namespace vc {

constexpr size_t F_THIN_COMMIT_BYTES = 2 * (size_t)FT * 16;

// LPG = lanes per gate (1 or 4).  With at most F_WORKERS / 4 gates per CTA a gate is spread over four neighbouring lanes: after the
// challenge arrives each lane does ONE of the four multiplies that depend on it (fold lo, fold hi, W update, P update),
// the results are exchanged by shuffles, and lanes 0 and 1 do one product each — the chain from challenge to commit
// is two multiplies deep on every lane instead of five multiplies issued by one.  All lanes run the same instruction
// stream (operands are selected, not branched on); gates beyond ng mirror the last gate and commit nothing.  (Two lanes per gate
// for up to F_WORKERS / 2 gates was measured and is slower than one: 71.3 against 67.2 us on config 2's layer 15.)
template <int LPG>
__device__ __forceinline__ void thin_layer(const FusedArgs &a, FusedCtx &cx, const uint64_t *invfact, const uint32_t *pas,
                                           uint8_t *dyn, uint32_t layer, uint64_t *tr) {
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, G = gridDim.x, b = blockIdx.x;
    const LayerPlan &Lp = a.L[layer];
    const uint32_t si = Lp.log_n, s = a.L[layer + 1].log_n;
    const bool has_ign = Lp.has_relay != 0;
    const uint64_t *__restrict__ Vb = a.L[layer + 1].V;
    const CtaPlan cp = Lp.cta[b];
    const uint32_t g0 = cp.g0, ng = cp.g1 - cp.g0;           // ng <= F_WORKERS
    const uint32_t q = LPG == 1 ? 0 : tid & (LPG - 1), gi = LPG == 4 ? tid >> 2 : tid;
    const bool live = gi < ng;                               // this lane's gate exists
    constexpr uint32_t GPW = 32 / LPG;                       // gates per warp
    const bool act = LPG == 1 ? live : gi < ((ng + GPW - 1) & ~(GPW - 1));   // uniform within a warp for LPG > 1
    const uint32_t g = g0 + (live ? gi : (ng ? ng - 1 : 0));
    ulonglong2 *cbuf = reinterpret_cast<ulonglong2 *>(dyn);   // [2][FT] committed products
    uint64_t *bufX = reinterpret_cast<uint64_t *>(dyn + Lp.off_tab), *bufY = bufX + Lp.xw;
    uint64_t *scr = reinterpret_cast<uint64_t *>(dyn + Lp.off_scr);
    const uint64_t seed = cx.seed;

    // ---- a3 + phase-1 state
    __syncthreads();
    VC_TR(30);
    uint32_t ctr = (uint32_t)cx.ctr;
    uint32_t i1 = 0, i2 = 0, t = VC_RELAY, idx = 0;
    uint64_t W = 0, cP = fp61::P, P = 0;             // P: the plain weight beta(z,g) eq(low bits of in1[g], r1[0..j)), tracked in phase 1
    uint64_t other = 0;
    if (act) {                                       // the gate's record and fixed operand travel while the eq table is built
        Wires(Lp, &cx.wrule).get(g, i1, i2, t);
        other = __ldg(Vb + i2);
    }
    const EqTab eb = build_eq_tab(bufX, bufX + (1u << F_EQLOG), scr, cx.z, si, tid, FT);
    __syncthreads();
    VC_TR(31);
    if (act) {
        P = eb.eq_of(g);
        uint64_t c; uint32_t ign;
        gate_state(1, t, P, other, W, c, ign);
        cP = c + fp61::P; idx = i1;
    }
    if (layer == 0) {                                // a2: start claim V~_0(z_0) = sum_g beta(z_0,g) V_0[g]
        uint64_t part = (live && q == 0) ? fp61::mul(eb.eq_of(g), __ldg(Lp.V + g)) : 0;
        part = warp_sum61(part);
        if (lane == 0) cx.red[warp * 4] = part;
        __syncthreads();
        if (warp == 0) { const uint64_t t0 = warp_sum61(lane < (uint32_t)FT / 32 ? cx.red[lane * 4] : 0); if (lane == 0) cx.acc[0] = t0; }
        grid_allreduce(cx, a, 1, false);
        if (tid == 0) cx.claim = cx.acc[0];
    }
    VC_TR(32);
    __syncthreads();
    VC_TR(33);
    uint32_t ep = cx.epoch, par = 0;
    RoundPend pd; pd.tr1 = pd.tr2 = nullptr; pd.s1 = pd.s2 = 0;

    for (int ph = 0; ph < 2; ph++) {
        const uint32_t K = Lp.K[ph], blo = cp.blo[ph], nbk = cp.nb[ph];
        uint64_t *rr = ph == 0 ? cx.r1 : cx.r2;
        if (ph == 1) {                               // phase switch: P = beta(z,g) eq(in1[g], r1) is in the register; the phase-2 state
            VC_TR(34);
            __syncthreads();                         // v1 and r1[s-1] are visible
            VC_TR(35);
            if (act) {
                P = fp61::mul(P, ((i1 >> (s - 1)) & 1u) ? cx.r1[s - 1] : fp61::sub(1, cx.r1[s - 1]));   // the last factor of phase 1
                uint64_t c; uint32_t ign;
                gate_state(2, t, P, cx.v1, W, c, ign);
                cP = c + fp61::P; idx = i2 | (ign << 31);
            }
            VC_TR(37);
        }
        uint64_t r_prev = 0;
        for (uint32_t j = 0; j < s; j++) {
            bool fence = false;
            if (K >= 2 && j == K - 1) {              // publish level K-1 (read by round K's gates and by its level build)
                if (Lp.pub_slice[ph]) {              // the slices cover the level: fold this CTA's share from level K-2 of its slice
                    __syncthreads();                 // level K-2 (built in the shadow of the last rendezvous) and r_prev are in place
                    const uint32_t o0 = cp.own_lo[ph], on = cp.own_n[ph];
                    for (uint32_t e = tid; e < on; e += FT) {
                        const uint32_t idx = o0 + e;
                        uint64_t x0, x1;
                        if (K == 2) { const ulonglong2 p = __ldg(reinterpret_cast<const ulonglong2 *>(Vb + 2 * (size_t)idx)); x0 = p.x; x1 = p.y; }
                        else {
                            const uint64_t *src = ((K - 2) & 1) ? bufX : bufY;
                            const ulonglong2 p = *reinterpret_cast<const ulonglong2 *>(src + (2 * (size_t)idx - ((size_t)blo << 2)));
                            x0 = p.x; x1 = p.y;
                        }
                        __stcg(a.Tg + idx, fold2(x0, x1, r_prev));
                    }
                } else {
                    const uint32_t E = 1u << (s - K + 1);
                    publish_level(Vb, rr, K - 1, (uint32_t)(((uint64_t)b * E) / G), (uint32_t)(((uint64_t)(b + 1) * E) / G), scr, a.Tg);
                }
                fence = true;
            }
            // ---- a4 for this thread's gate, against level j-1 folded on the fly (level 0 in round 0)
            if (act) {
                const uint32_t bit = (idx >> j) & 1u, u = (idx & F_IDX_MASK) >> (j + 1);
                uint64_t lo, hi;
                if (j == 0) {
                    const ulonglong2 p = *reinterpret_cast<const ulonglong2 *>(Vb + 2 * (size_t)u);
                    lo = p.x; hi = p.y;
                } else {
                    ulonglong2 q0, q1;
                    if (j == 1) {
                        q0 = *reinterpret_cast<const ulonglong2 *>(Vb + 4 * (size_t)u);
                        q1 = *reinterpret_cast<const ulonglong2 *>(Vb + 4 * (size_t)u + 2);
                    } else if (j == K) {
                        q0 = __ldcg(reinterpret_cast<const ulonglong2 *>(a.Tg + 4 * (size_t)u));
                        q1 = __ldcg(reinterpret_cast<const ulonglong2 *>(a.Tg + 4 * (size_t)u + 2));
                    } else {
                        const uint64_t *src = ((j - 1) & 1) ? bufX : bufY;
                        const uint32_t base = (j - 1 < K) ? blo << (K - j + 1) : 0;
                        q0 = *reinterpret_cast<const ulonglong2 *>(src + (4 * (size_t)u - base));
                        q1 = *reinterpret_cast<const ulonglong2 *>(src + (4 * (size_t)u - base) + 2);
                    }
                    const uint64_t fj = ((idx >> (j - 1)) & 1u) ? r_prev : fp61::sub(1, r_prev);
                    if (LPG == 4) {
                        // lane 0: lo = x0 + r (x1 - x0) of the first pair, lane 1: hi of the second, lane 2: W fj, lane 3: P fj
                        const uint64_t x0 = q == 0 ? q0.x : q1.x, x1 = q == 0 ? q0.y : q1.y;
                        const uint64_t ma = q < 2 ? r_prev : (q == 2 ? W : P), mb_ = q < 2 ? fp61::sub(x1, x0) : fj;
                        const uint64_t pr = fp61::mul(ma, mb_), val = q < 2 ? fp61::add(x0, pr) : pr;
                        const uint32_t l4 = lane & ~3u;
                        lo = __shfl_sync(0xffffffffu, val, l4); hi = __shfl_sync(0xffffffffu, val, l4 + 1);
                        W = __shfl_sync(0xffffffffu, val, l4 + 2);
                        const uint64_t Pn = __shfl_sync(0xffffffffu, val, l4 + 3);
                        if (ph == 0) P = Pn;
                    } else {
                        lo = fold2(q0.x, q0.y, r_prev); hi = fold2(q1.x, q1.y, r_prev);
                        W = fp61::mul(W, fj);
                        if (ph == 0) P = fp61::mul(P, fj);   // off the products' chain: spares two eq tables at the phase switch
                    }
                }
                if (has_ign && (idx >> 31)) { lo = 0; hi = 0; }
                const uint64_t mb = (bit ? hi : lo) + cP, m2 = 2 * hi + cP - lo;
                if (LPG > 1) {                       // lane 0: W (x_b + c) with the bit, lane 1: W (x_2 + c)
                    const uint64_t m = q == 0 ? mb : m2;
                    const uint64_t pr = fp61::fold128(fp61::mulhi(W, m), W * m) | (q == 0 ? (uint64_t)bit << 63 : 0);
                    if (live && q < 2) reinterpret_cast<uint64_t *>(cbuf + par * FT + gi)[q] = pr;
                } else {
                    ulonglong2 o;
                    o.x = fp61::fold128(fp61::mulhi(W, mb), W * mb) | ((uint64_t)bit << 63);
                    o.y = fp61::fold128(fp61::mulhi(W, m2), W * m2);
                    cbuf[par * FT + tid] = o;
                }
            }
            VC_TR(41);
            __syncthreads();                         // every contribution of this CTA to message j is committed
            VC_TR(42);
            uint64_t *rslot = rr + j;
            if (warp == 15) {
                // ---- a5, off the critical path: sum the committed products, add them to the round's data words
                const ulonglong2 *cb = cbuf + par * FT;
                uint64_t Sl = 0, S1l = 0, Tl = 0, T1l = 0; uint32_t Sh = 0, S1h = 0, Th = 0, T1h = 0;
                for (uint32_t i = lane; i < ng; i += 32) {
                    const ulonglong2 q = cb[i];
                    const uint32_t bit = (uint32_t)(q.x >> 63);
                    const uint64_t v1 = q.x & ~(1ull << 63);
                    add_c(Sl, Sh, v1, 1u); add_c(S1l, S1h, v1, bit);
                    add_c(Tl, Th, q.y, 1u); add_c(T1l, T1h, q.y, bit);
                }
                const uint64_t x = fp61::fold128(Sh, Sl), x1 = fp61::fold128(S1h, S1l), y = fp61::fold128(Th, Tl), y1 = fp61::fold128(T1h, T1l);
                const uint64_t t0 = warp_sum61(fp61::sub(x, x1)), t1 = warp_sum61(x1);
                const uint64_t t2 = warp_sum61(fp61::sub(fp61::add(fp61::dbl(y1), y1), y));
                reducer_post(a, ep, t0, t1, t2, tr, pd);
            } else {
                if (warp == 0) {                     // ---- the rendezvous: count word only
                    round_rendezvous(a, ep, fence, rslot, seed, ctr);
                } else if (j >= 1 && j + 1 != K) {   // ---- warps 1..14: build level j in the shadow of the wait
                    const uint32_t wt = tid - 32, WT = F_WORKERS - 32;
                    uint64_t *dst = (j & 1) ? bufX : bufY;
                    const uint64_t *prev = (j & 1) ? bufY : bufX;
                    const bool slice = j < K;
                    const uint32_t cnt = slice ? nbk << (K - j) : 1u << (s - j);
                    if (j == 1 || j == K) {
                        const uint64_t *src = j == 1 ? Vb + (slice ? (size_t)blo << K : 0) : a.Tg;
                        for (uint32_t v = wt; v < cnt; v += WT) {
                            const ulonglong2 p = __ldcg(reinterpret_cast<const ulonglong2 *>(src + 2 * (size_t)v));
                            dst[v] = fold2(p.x, p.y, r_prev);
                        }
                    } else {
                        for (uint32_t v = wt; v < cnt; v += WT) dst[v] = fold2(prev[2 * v], prev[2 * v + 1], r_prev);
                    }
                }
                VC_TR(43);
                bar_workers();
                VC_TR(44);
            }
            r_prev = *rslot;                         // (the reducer never uses it)
            ctr++; tr += 3; ep++; par ^= 1;
        }
        // ---- V~_{i+1}(r) = the two entries of level s-1 folded with the last challenge
        if (tid == 0) {
            const uint64_t *t1 = s == 1 ? Vb : (((s - 1) & 1) ? bufX : bufY);
            const uint64_t val = fold2(t1[0], t1[1], r_prev);
            if (ph == 0) cx.v1 = val; else cx.v2 = val;
        }
    }
    if (tid == 0) { cx.ctr = ctr; cx.epoch = ep; }
    __syncthreads();
    VC_TR(17);
    // ---- a7: line restriction, all CTAs share the pass over V_{i+1}; the reducer converts the last two rounds'
    // messages into transcript words beside it (their slots are not touched by the all-reduce below: ring of 8)
    if (s > 1) {
        const uint32_t ltb = fused_line_tb_grid(s, FT), lthr = (1u << ltb) > 32 ? (1u << ltb) : 32;
        if (tid < lthr) line_partials(Vb, s, cx, pas, reinterpret_cast<uint64_t *>(dyn), b, G, tid, lthr, ltb);
        if (warp == 15) reducer_flush(a, pd);        // lthr <= 2^7 on this path: warp 15 is never in line_partials
        grid_allreduce(cx, a, s - 1, false);
    } else if (warp == 15) reducer_flush(a, pd);
    VC_TR(18);
    line_finish(s, cx, invfact, tr, b == 0, tid);
    __syncthreads();
    VC_TR(19);
}

}  // namespace vc
