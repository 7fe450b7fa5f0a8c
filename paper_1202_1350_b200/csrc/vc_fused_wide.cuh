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
#include <type_traits>

#include "vc_fused.cuh"
#include "vc_fused_line.cuh"
#include "vc_fused_small.cuh"

namespace vc {

// level K-1 of the fold table, entries [e0, e1): T[e] = sum_v eq(v, rr[0..K-1)) V[e 2^(K-1) + v].  One warp per entry.
__device__ __noinline__ void publish_level(const uint64_t *__restrict__ Vb, const uint64_t *rr, uint32_t km1, uint32_t e0,
                                              uint32_t e1, uint64_t *eqt, uint64_t *Tg) {
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    __syncthreads();                                             // rr[km1-1] (written by the last rendezvous) is visible
    if (km1 <= 5) {                                              // 2^km1 lanes per entry: no table, no further barrier
        const uint32_t gs = 1u << km1, per = 32u >> km1, sub = lane & (gs - 1), ent = lane >> km1;
        const uint64_t w = eq_direct(sub, rr, 0, km1);
        for (uint32_t ew = e0 + warp * per; ew < e1; ew += (FT / 32) * per) {
            const uint32_t e = ew + ent;
            uint64_t v = e < e1 ? fp61::mul(w, __ldg(Vb + ((size_t)e << km1) + sub)) : 0;
            for (uint32_t off = gs >> 1; off; off >>= 1) v = fp61::add(v, __shfl_xor_sync(0xffffffffu, v, off));
            if (sub == 0 && e < e1) __stcg(Tg + e, v);
        }
        return;
    }
    build_eq10(eqt + 64, eqt, rr, 0, km1, tid, FT);              // eqt[0..64): the two 5-variable factors
    __syncthreads();
    eqt += 64;
    for (uint32_t e = e0 + warp; e < e1; e += FT / 32) {
        const uint64_t *src = Vb + ((size_t)e << km1);
        acc128 A; A.clear();
        uint64_t sum = 0;
        const uint32_t nv = 1u << km1;
        for (uint32_t v0 = lane; v0 < nv; v0 += 32 * 8) {        // 8 loads in flight per lane, then 8 products
            uint64_t w[8];
#pragma unroll
            for (int q = 0; q < 8; q++) w[q] = v0 + 32 * q < nv ? __ldg(src + v0 + 32 * q) : 0;
#pragma unroll
            for (int q = 0; q < 8; q++) if (v0 + 32 * q < nv) A.mac(eqt[v0 + 32 * q], w[q]);
            sum = fp61::add(sum, A.value()); A.clear();
        }
        sum = warp_sum61(sum);
        if (lane == 0) __stcg(Tg + e, sum);
    }
}

// dst[v] = fold(src[2v], src[2v+1]; r), v < cnt, src in global memory (read-only); 4 loads in flight per thread
__device__ __noinline__ void fold_level_from_global(uint64_t *dst, const uint64_t *src, uint32_t cnt, uint64_t r, uint32_t t,
                                                    uint32_t nthr) {
    for (uint32_t v0 = t; v0 < cnt; v0 += 4 * nthr) {
        ulonglong2 p[4];
#pragma unroll
        for (int q = 0; q < 4; q++)
            if (v0 + q * nthr < cnt) p[q] = __ldg(reinterpret_cast<const ulonglong2 *>(src + 2 * (size_t)(v0 + q * nthr)));
#pragma unroll
        for (int q = 0; q < 4; q++)
            if (v0 + q * nthr < cnt) dst[v0 + q * nthr] = fold2(p[q].x, p[q].y, r);
    }
}

// One resident gate against a shared-memory (or level-0 global) table: pending weight update, then the two products.
// cP = c + p is what the state holds (any representative of c works as an addend; this one saves the "+ p").
struct GateIn { uint64_t W, cP; uint32_t idx; };
__device__ __forceinline__ void gate_apply(GateIn &gi, const ulonglong2 pr, uint32_t j, bool upd, uint64_t r_prev, uint64_t omr,
                                           bool has_ign, acc128 &X, acc128 &X1, acc128 &Y, acc128 &Y1) {
    if (upd) gi.W = fp61::mul(gi.W, ((gi.idx >> (j - 1)) & 1u) ? r_prev : omr);
    uint64_t lo = pr.x, hi = pr.y;
    if (has_ign && (gi.idx >> 31)) { lo = 0; hi = 0; }
    const uint32_t bit = (gi.idx >> j) & 1u;
    const uint64_t mb = (bit ? hi : lo) + gi.cP;                 // < 2^61 + 2^62
    const uint64_t m2 = 2 * hi + gi.cP - lo;                     // 2 hi - lo + c + p  in (0, 2^63.4)
    fp61::mac2(X.lo, X.hi, X1.lo, X1.hi, gi.W, mb, bit);
    fp61::mac2(Y.lo, Y.hi, Y1.lo, Y1.hi, gi.W, m2, bit);
}

// (lo,hi) += a*b
__device__ __forceinline__ void mac1(acc128 &A, uint64_t pl, uint64_t ph) {
    asm("add.cc.u64 %0, %0, %2;\n\taddc.u64 %1, %1, %3;" : "+l"(A.lo), "+l"(A.hi) : "l"(pl), "l"(ph));
}
// The resident hot loop: this thread's gates l = k GT + tid (k < nmine) against the level-j table `tb` (already offset
// by the slice base), two gates in flight.  Accumulators per bit value: X0/X1 collect W (x_b + c), Y0/Y1 collect
// W (x_2 + c); G[0] = X0, G[1] = X1, G[2] = 2 Y1 - Y0.  s4 receives the canonical sums (flushed every 8 products).
template <bool IGN>
__device__ __forceinline__ void hot_gates(const bool UPD, uint64_t *sW, const uint64_t *sC, const uint32_t *sI,
                                          const uint64_t *tb, uint32_t j, uint32_t nmine, uint32_t tid, uint64_t r_prev,
                                          uint64_t omr, uint64_t (&s4)[4]) {
    constexpr uint32_t GT = FT;                  // all sixteen warps own gates on this path
    acc128 X0, X1, Y0, Y1; X0.clear(); X1.clear(); Y0.clear(); Y1.clear();
    const uint32_t sh = j + 1;
    auto one = [&](uint64_t &W, uint64_t cP, uint32_t idx, const ulonglong2 pr) {
        if (UPD) W = fp61::mul(W, ((idx >> (j - 1)) & 1u) ? r_prev : omr);
        uint64_t lo = pr.x, hi = pr.y;
        if (IGN && (idx >> 31)) { lo = 0; hi = 0; }
        const uint32_t bit = (idx >> j) & 1u;
        const uint64_t mb = (bit ? hi : lo) + cP;                // < 2^61 + 2^62
        const uint64_t m2 = 2 * hi + cP - lo;                    // 2 hi - lo + c + p  in (0, 2^63)
        const uint64_t pl = W * mb, ph = fp61::mulhi(W, mb), ql = W * m2, qh = fp61::mulhi(W, m2);
        if (bit) { mac1(X1, pl, ph); mac1(Y1, ql, qh); } else { mac1(X0, pl, ph); mac1(Y0, ql, qh); }
    };
    auto flush = [&]() {
        s4[0] = fp61::add(s4[0], X0.value()); s4[1] = fp61::add(s4[1], X1.value());
        s4[2] = fp61::add(s4[2], Y0.value()); s4[3] = fp61::add(s4[3], Y1.value());
        X0.clear(); X1.clear(); Y0.clear(); Y1.clear();
    };
    uint32_t k = 0;
    for (; k + 2 <= nmine; k += 2) {
        const uint32_t l0 = k * GT + tid, l1 = l0 + GT;
        uint64_t Wa = sW[l0], Wb = sW[l1];
        const uint64_t ca = sC[l0], cb = sC[l1];
        const uint32_t ia = sI[l0], ib = sI[l1];
        const ulonglong2 pa = *reinterpret_cast<const ulonglong2 *>(tb + 2 * (size_t)((ia & F_IDX_MASK) >> sh));
        const ulonglong2 pb = *reinterpret_cast<const ulonglong2 *>(tb + 2 * (size_t)((ib & F_IDX_MASK) >> sh));
        one(Wa, ca, ia, pa);
        one(Wb, cb, ib, pb);
        if (UPD) { sW[l0] = Wa; sW[l1] = Wb; }
        if ((k & 6) == 6) flush();                               // 8 products per accumulator at most
    }
    if (k < nmine) {
        const uint32_t l0 = k * GT + tid;
        uint64_t Wa = sW[l0];
        const uint32_t ia = sI[l0];
        const ulonglong2 pa = *reinterpret_cast<const ulonglong2 *>(tb + 2 * (size_t)((ia & F_IDX_MASK) >> sh));
        one(Wa, sC[l0], ia, pa);
        if (UPD) sW[l0] = Wa;
    }
    flush();
}

// ---- the resident hot loop for rounds j >= 1 of a sliced phase: table in shared memory, weight update pending.
// Per gate-round: one multiply for the weight, two products into 128-bit accumulators, nothing else that is not a load
// or an address.  Against hot_gates it drops (a) the canonical form of W between rounds: W' = W f is left below
// 2^61 + 4 (w1 <= 2^29 keeps every partial product in range: p11 = w1 f1 < 2^58, mid = w0 f1 + w1 f0 < 2^62), and the
// fold uses 2^61 = 1: W f = p00 + mid 2^32 + p11 2^64 = (p00 mod') + (mid >> 29) + (mid & (2^29-1)) 2^32 + 8 p11, with
// 8 f1 formed once per gate from the selected f; (b) generic addressing: the table is addressed as shared memory;
// (c) the accumulator flushes: products are < 2^61.01 * 2^63, fifteen of them fit 128 bits, so one flush per 14 gates.
__device__ __forceinline__ uint64_t mul_wide(uint32_t a, uint32_t b) { uint64_t r; asm("mul.wide.u32 %0, %1, %2;" : "=l"(r) : "r"(a), "r"(b)); return r; }
__device__ __forceinline__ uint64_t mad_wide(uint32_t a, uint32_t b, uint64_t c) { uint64_t r; asm("mad.wide.u32 %0, %1, %2, %3;" : "=l"(r) : "r"(a), "r"(b), "l"(c)); return r; }
__device__ __forceinline__ uint64_t mul_lazy61(uint64_t W, uint32_t f0, uint32_t f1) {
    const uint32_t w0 = (uint32_t)W, w1 = (uint32_t)(W >> 32), f1x8 = f1 << 3;
    const uint64_t p00 = mul_wide(w0, f0);
    const uint64_t mid = mad_wide(w1, f0, mul_wide(w0, f1));                              // < 2^62
    uint64_t s = mad_wide(w1, f1x8, mid >> 29);                                             // 8 p11 + (mid >> 29) < 2^61 + 2^33
    s = ((uint64_t)((uint32_t)(s >> 32) + ((uint32_t)mid & 0x1fffffffu)) << 32) | (uint32_t)s;   // + (mid & (2^29-1)) 2^32: high word only, < 2^62
    s += (p00 & fp61::P) + (p00 >> 61);                                                     // < 2^63
    return (s & fp61::P) + (s >> 61);                                                       // < 2^61 + 4
}
__device__ __forceinline__ ulonglong2 lds_pair(uint32_t saddr) {
    ulonglong2 v;
    asm volatile("ld.shared.v2.u64 {%0, %1}, [%2];" : "=l"(v.x), "=l"(v.y) : "r"(saddr));
    return v;
}
#ifndef VC_HOT_ILP
#define VC_HOT_ILP 2
#endif
template <bool IGN>
__device__ __forceinline__ void hot_gates_sm(uint64_t *sW, const uint64_t *sC, const uint32_t *sI, uint32_t tb_s, uint32_t j,
                                             uint32_t nmine, uint32_t tid, uint64_t r_prev, uint64_t omr, uint64_t (&s4)[4]) {
    constexpr uint32_t GT = FT, CHUNK = 14;
    acc128 X0, X1, Y0, Y1; X0.clear(); X1.clear(); Y0.clear(); Y1.clear();
    const uint32_t sh = j + 1;
    const uint32_t r0 = (uint32_t)r_prev, r1 = (uint32_t)(r_prev >> 32), o0 = (uint32_t)omr, o1 = (uint32_t)(omr >> 32);
    auto one = [&](uint64_t &W, uint64_t cP, uint32_t idx, const ulonglong2 pr) {
        const bool bp = (idx >> (j - 1)) & 1u;
        W = mul_lazy61(W, bp ? r0 : o0, bp ? r1 : o1);
        uint64_t lo = pr.x, hi = pr.y;
        if (IGN && (idx >> 31)) { lo = 0; hi = 0; }
        const uint32_t bit = (idx >> j) & 1u;
        const uint64_t mb = (bit ? hi : lo) + cP;                // < 2^61 + 2^62
        const uint64_t m2 = 2 * hi + cP - lo;                    // 2 hi - lo + c + p  in (0, 2^63)
        const uint64_t pl = W * mb, ph = fp61::mulhi(W, mb), ql = W * m2, qh = fp61::mulhi(W, m2);
        if (bit) { mac1(X1, pl, ph); mac1(Y1, ql, qh); } else { mac1(X0, pl, ph); mac1(Y0, ql, qh); }
    };
    auto flush = [&]() {
        s4[0] = fp61::add(s4[0], X0.value()); s4[1] = fp61::add(s4[1], X1.value());
        s4[2] = fp61::add(s4[2], Y0.value()); s4[3] = fp61::add(s4[3], Y1.value());
        X0.clear(); X1.clear(); Y0.clear(); Y1.clear();
    };
    uint32_t k = 0, inacc = 0;
#if VC_HOT_ILP == 4
    for (; k + 4 <= nmine; k += 4) {
        const uint32_t l0 = k * GT + tid, l1 = l0 + GT, l2 = l1 + GT, l3 = l2 + GT;
        uint64_t Wa = sW[l0], Wb = sW[l1], Wc = sW[l2], Wd = sW[l3];
        const uint64_t ca = sC[l0], cb = sC[l1], cc = sC[l2], cd = sC[l3];
        const uint32_t ia = sI[l0], ib = sI[l1], ic = sI[l2], id = sI[l3];
        const ulonglong2 pa = lds_pair(tb_s + (((IGN ? ia & F_IDX_MASK : ia) >> sh) << 4));
        const ulonglong2 pb = lds_pair(tb_s + (((IGN ? ib & F_IDX_MASK : ib) >> sh) << 4));
        const ulonglong2 pc = lds_pair(tb_s + (((IGN ? ic & F_IDX_MASK : ic) >> sh) << 4));
        const ulonglong2 pd = lds_pair(tb_s + (((IGN ? id & F_IDX_MASK : id) >> sh) << 4));
        one(Wa, ca, ia, pa); one(Wb, cb, ib, pb); one(Wc, cc, ic, pc); one(Wd, cd, id, pd);
        sW[l0] = Wa; sW[l1] = Wb; sW[l2] = Wc; sW[l3] = Wd;
        inacc += 4;
        if (inacc >= CHUNK - 2) { flush(); inacc = 0; }
    }
#endif
    for (; k + 2 <= nmine; k += 2) {
        const uint32_t l0 = k * GT + tid, l1 = l0 + GT;
        uint64_t Wa = sW[l0], Wb = sW[l1];
        const uint64_t ca = sC[l0], cb = sC[l1];
        const uint32_t ia = sI[l0], ib = sI[l1];
        const ulonglong2 pa = lds_pair(tb_s + (((IGN ? ia & F_IDX_MASK : ia) >> sh) << 4));
        const ulonglong2 pb = lds_pair(tb_s + (((IGN ? ib & F_IDX_MASK : ib) >> sh) << 4));
        one(Wa, ca, ia, pa);
        one(Wb, cb, ib, pb);
        sW[l0] = Wa; sW[l1] = Wb;
        inacc += 2;
        if (inacc >= CHUNK) { flush(); inacc = 0; }
    }
    if (k < nmine) {
        const uint32_t l0 = k * GT + tid;
        uint64_t Wa = sW[l0];
        const uint32_t ia = sI[l0];
        const ulonglong2 pa = lds_pair(tb_s + (((IGN ? ia & F_IDX_MASK : ia) >> sh) << 4));
        one(Wa, sC[l0], ia, pa);
        sW[l0] = Wa;
    }
    flush();
}

__device__ __forceinline__ void wide_layer(const FusedArgs &a, FusedCtx &cx, const uint64_t *invfact, const uint32_t *pas, uint8_t *dyn,
                                           uint32_t layer, uint64_t *tr) {
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, G = gridDim.x, b = blockIdx.x;
    const LayerPlan &Lp = a.L[layer];
    const uint32_t si = Lp.log_n, s = a.L[layer + 1].log_n;
    const bool res = Lp.resident != 0, has_ign = Lp.has_relay != 0;
    const uint64_t *__restrict__ Vb = a.L[layer + 1].V;
    const CtaPlan cp = Lp.cta[b];
    const uint32_t g0 = cp.g0, ng = cp.g1 - cp.g0;
    const uint32_t nk = (ng + FT - 1) / FT;
    constexpr uint32_t GT = FT;                  // all sixteen warps own gates: l = k GT + tid.  Between the commit barrier and the
    // challenge warp 0 runs the rendezvous, warp 15 sums the committed words into the round's data words and warp 14 keeps
    // the transcript (CTA 0) / recycles slots (last CTA): the three jobs share the rendezvous' latency
    const uint32_t nmine = tid < ng ? (ng - tid + GT - 1) / GT : 0;
    ulonglong2 *cbuf = reinterpret_cast<ulonglong2 *>(dyn + Lp.off_commit);       // [GT][2]: X, X1, Y, Y1 sums per worker
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
    const EqTab eb = build_eq_tab(bufX, bufX + (1u << F_EQLOG), scr, cx.z, si, tid, FT);
    __syncthreads();
    uint64_t claim_part = 0;
    auto setup1 = [&](auto resident) {
        const Wires wr(Lp, &cx.wrule);                      // records, or the rule that replaces them (built outside the loop: Lp sits in global memory)
#pragma unroll 2
        for (uint32_t k = 0; k < nk; k++) {
            const uint32_t l = k * FT + tid;
            const bool valid = l < ng;
            const uint32_t g = valid ? g0 + l : g0;
            uint32_t i1, i2, t;
            wr.get(g, i1, i2, t);
            const uint64_t other = __ldg(Vb + i2);
            const uint64_t P = eb.eq_of(g);
            uint64_t W, c; uint32_t ign;
            gate_state(1, t, P, other, W, c, ign);
            if (valid) {
                if (decltype(resident)::value) { sW[l] = W; sC[l] = c + fp61::P; sI[l] = i1; } else { a.P[g] = W; a.C[g] = c + fp61::P; }
                if (layer == 0) claim_part = fp61::add(claim_part, fp61::mul(P, __ldg(Lp.V + g)));
            }
        }
    };
    if (res) setup1(std::true_type{}); else setup1(std::false_type{});
    if (layer == 0) {                            // a2: start claim V~_0(z_0) = sum_g beta(z_0,g) V_0[g]
        claim_part = warp_sum61(claim_part);
        if (lane == 0) cx.red[warp * 4] = claim_part;
        __syncthreads();
        if (warp == 0) { const uint64_t t0 = warp_sum61(lane < (uint32_t)FT / 32 ? cx.red[lane * 4] : 0); if (lane == 0) cx.acc[0] = t0; }
        grid_allreduce(cx, a, 1, false);
        if (tid == 0) cx.claim = cx.acc[0];
    }

    VC_TR(11);
    __syncthreads();
    uint32_t ep = cx.epoch;
    RoundPend pd; pd.tr1 = pd.tr2 = nullptr; pd.s1 = pd.s2 = 0;
    for (int ph = 0; ph < 2; ph++) {
        const uint32_t mode = Lp.mode[ph], K = Lp.K[ph], blo = cp.blo[ph], nbk = cp.nb[ph];
        uint64_t *rr = ph == 0 ? cx.r1 : cx.r2;
        if (ph == 1) {
            // ---- phase switch: plain weight P = beta(z,g) eq(in1[g], r1), then the phase-2 state
            __syncthreads();                     // v1, r1[s-1] visible; phase-1 tables dead
            const uint64_t v1 = cx.v1;
            const EqTab e0 = build_eq_tab(bufX, bufX + (1u << F_EQLOG), scr, cx.z, si, tid, FT);
            const EqTab e1 = build_eq_tab(bufX + (2u << F_EQLOG), bufX + (3u << F_EQLOG), scr + 128, cx.r1, s, tid, FT);
            __syncthreads();
            auto setup2 = [&](auto resident) {
                const Wires wr(Lp, &cx.wrule);
#pragma unroll 2
                for (uint32_t k = 0; k < nk; k++) {
                    const uint32_t l = k * FT + tid;
                    const bool valid = l < ng;
                    const uint32_t g = valid ? g0 + l : g0;
                    uint32_t i1, i2, t;
            wr.get(g, i1, i2, t);
                    const uint64_t P = fp61::mul(e0.eq_of(g), e1.eq_of(i1));
                    uint64_t W, c; uint32_t ign;
                    gate_state(2, t, P, v1, W, c, ign);
                    if (valid) {
                        if (decltype(resident)::value) { sW[l] = W; sC[l] = c + fp61::P; sI[l] = i2 | (ign << 31); }
                        else { a.P[g] = W; a.C[g] = c + fp61::P; }
                    }
                }
            };
            if (res) setup2(std::true_type{}); else setup2(std::false_type{});
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
                            fold_level_from_global(dst, src, cnt, r_prev, tid, GT);
                        } else {
                            for (uint32_t v = tid; v < cnt; v += GT) dst[v] = fold2(prev[2 * v], prev[2 * v + 1], r_prev);
                        }
                        base = blo << (K - j);
                    } else {                     // the whole table: from the published level K-1 (j = K >= 2), from V (j = 1),
                        const uint32_t cnt = 1u << (s - j);                         // else from the previous buffer
                        if (j == 1 || j == K) {
                            const uint64_t *src = j == 1 ? Vb : a.Tg;
                            for (uint32_t v = tid; v < cnt; v += GT) {
                                const ulonglong2 p = __ldcg(reinterpret_cast<const ulonglong2 *>(src + 2 * (size_t)v));
                                dst[v] = fold2(p.x, p.y, r_prev);
                            }
                        } else {
                            for (uint32_t v = tid; v < cnt; v += GT) dst[v] = fold2(prev[2 * v], prev[2 * v + 1], r_prev);
                        }
                    }
                    tab = dst;
                }
                if (K >= 2 && j == K - 1) {      // publish level K-1 for the next round (needs r_0..r_{K-2})
                    if (Lp.pub_slice[ph]) {      // the slices cover the level: this CTA's share is in the slice it has just folded
                        __syncthreads();
                        const uint64_t *lvl = (j & 1) ? bufX : bufY;
                        const uint32_t o0 = cp.own_lo[ph], on = cp.own_n[ph], sb0 = blo << 1;
                        for (uint32_t e = tid; e < on; e += GT) __stcg(a.Tg + o0 + e, lvl[o0 + e - sb0]);
                    } else {
                        const uint32_t E = 1u << (s - K + 1);
                        publish_level(Vb, rr, K - 1, (uint32_t)(((uint64_t)b * E) / G), (uint32_t)(((uint64_t)(b + 1) * E) / G), scr, a.Tg);
                    }
                    fence = true;
                }
            } else {                             // GLOBAL: materialise level j (j >= 1) for the next round's on-the-fly fold
                tab = j <= 1 ? Vb : ((j & 1) ? a.T1 : a.T0);                       // level j-1
                if (j >= 1) {
                    uint64_t *Aout = (j & 1) ? a.T0 : a.T1;                          // level j
                    const uint32_t cnt = 1u << (s - j);
                    for (uint32_t v = b * GT + tid; v < cnt; v += G * GT) {
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
            {
                const uint64_t omr = fp61::sub(1, r_prev);
                const bool upd = j >= 1;
                acc128 X, X1, Y, Y1; X.clear(); X1.clear(); Y.clear(); Y1.clear();
                uint64_t s4[4] = {0, 0, 0, 0};                 // canonical running sums of X, X1, Y, Y1 (flushed every 8 products)
                if (res && mode == F_MODE_SLICE) {
                    // hot loop: state in shared memory; the table is level 0 in L2 (round 0) or a shared-memory buffer
                    if (j >= 1) {                          // level j sits in shared memory and a weight update is pending: the slim loop
                        const uint32_t tb_s = (uint32_t)__cvta_generic_to_shared(tab) - base * 8u;
                        if (has_ign) hot_gates_sm<true>(sW, sC, sI, tb_s, j, nmine, tid, r_prev, omr, s4);
                        else hot_gates_sm<false>(sW, sC, sI, tb_s, j, nmine, tid, r_prev, omr, s4);
                    } else if (has_ign) hot_gates<true>(upd, sW, sC, sI, tab - base, j, nmine, tid, r_prev, omr, s4);
                    else hot_gates<false>(upd, sW, sC, sI, tab - base, j, nmine, tid, r_prev, omr, s4);
                } else {
                    const Wires wr(Lp, &cx.wrule);
                    for (uint32_t k = 0; k < nmine; k++) {
                        const uint32_t l = k * GT + tid, g = g0 + l;
                        GateIn A;
                        if (res) { A.W = sW[l]; A.cP = sC[l]; A.idx = sI[l]; }
                        else {
                            A.W = a.P[g]; A.cP = a.C[g];
                            if (wr.mode == W_GENERIC) A.idx = ph == 0 ? wr.in1[g] : (wr.in2[g] | ((wr.type[g] == VC_RELAY ? 1u : 0u) << 31));
                            else A.idx = ph == 0 ? wr.in1_of(g) : (wr.in2_of(g) | ((wr.type_of(g) == VC_RELAY ? 1u : 0u) << 31));
                        }
                        const uint32_t u = (A.idx & F_IDX_MASK) >> (j + 1);
                        ulonglong2 pr;
                        if (mode == F_MODE_SLICE || j == 0) {
                            pr = *reinterpret_cast<const ulonglong2 *>(tab + (2 * (size_t)u - base));
                        } else {                 // fold level j-1 on the fly with r_{j-1}
                            const ulonglong2 p0 = __ldcg(reinterpret_cast<const ulonglong2 *>(tab + 4 * (size_t)u));
                            const ulonglong2 p1 = __ldcg(reinterpret_cast<const ulonglong2 *>(tab + 4 * (size_t)u + 2));
                            pr.x = fold2(p0.x, p0.y, r_prev); pr.y = fold2(p1.x, p1.y, r_prev);
                        }
                        gate_apply(A, pr, j, upd, r_prev, omr, has_ign, X, X1, Y, Y1);
                        if (upd) { if (res) sW[l] = A.W; else a.P[g] = A.W; }
                        if ((k & 7) == 7) {
                            s4[0] = fp61::add(s4[0], X.value()); s4[1] = fp61::add(s4[1], X1.value());
                            s4[2] = fp61::add(s4[2], Y.value()); s4[3] = fp61::add(s4[3], Y1.value());
                            X.clear(); X1.clear(); Y.clear(); Y1.clear();
                        }
                    }
                    // totals -> per-bit sums: X0 = X - X1, Y0 = Y - Y1
                    s4[1] = fp61::add(s4[1], X1.value()); s4[3] = fp61::add(s4[3], Y1.value());
                    s4[0] = fp61::sub(fp61::add(s4[0], X.value()), s4[1]); s4[2] = fp61::sub(fp61::add(s4[2], Y.value()), s4[3]);
                }
                VC_TR(21);
                if (tid < ng) {                  // commit this worker's four canonical sums X0, X1, Y0, Y1
                    ulonglong2 o0, o1;
                    o0.x = s4[0]; o0.y = s4[1]; o1.x = s4[2]; o1.y = s4[3];
                    cbuf[2 * tid] = o0; cbuf[2 * tid + 1] = o1;
                }
            }
            VC_TR(15);
            __syncthreads();                     // every contribution of this CTA to message j is committed
            uint64_t *rslot = rr + j;
            if (warp == 15) {
                // ---- a5 in the shadow of the rendezvous: sum the committed words, add them to the round's data words
                const uint32_t nc = ng < GT ? ng : GT;
                uint64_t Sl = 0, S1l = 0, Tl = 0, T1l = 0; uint32_t Sh = 0, S1h = 0, Th = 0, T1h = 0;
                for (uint32_t i = lane; i < nc; i += 32) {
                    const ulonglong2 q0 = cbuf[2 * i], q1 = cbuf[2 * i + 1];
                    add_c(Sl, Sh, q0.x, 1u); add_c(S1l, S1h, q0.y, 1u); add_c(Tl, Th, q1.x, 1u); add_c(T1l, T1h, q1.y, 1u);
                }
                const uint64_t x = fp61::fold128(Sh, Sl), x1 = fp61::fold128(S1h, S1l), y = fp61::fold128(Th, Tl), y1 = fp61::fold128(T1h, T1l);
                const uint64_t t0 = warp_sum61(x), t1 = warp_sum61(x1);
                const uint64_t t2 = warp_sum61(fp61::sub(fp61::dbl(y1), y));        // x, y here are the bit-0 sums
                reducer_post_data(a, ep, t0, t1, t2);
            } else if (warp == 14) {
                reducer_housekeeping(a, ep, tr, pd);
            } else if (warp == 0) {
                round_rendezvous(a, ep, fence, rslot, seed, ctr);   // ---- a6: rendezvous, then the challenge
            }
            __syncthreads();
            VC_TR(16);
            ctr++; tr += 3; ep++;
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
    if (tid == 0) { cx.ctr = ctr; cx.epoch = ep; }
    if (warp == 14) reducer_flush(a, pd);                   // the last two rounds' messages
    __syncthreads();
    VC_TR(17);
    // ---- a7: line restriction, all CTAs share the pass over V_{i+1}
    if (s > 1) {
        const uint32_t ltb = fused_line_tb_grid(s, FT), lthr = (1u << ltb) > 32 ? (1u << ltb) : 32;
        if (tid < lthr) line_partials(Vb, s, cx, pas, reinterpret_cast<uint64_t *>(dyn), b, G, tid, lthr, ltb);
        grid_allreduce(cx, a, s - 1, false);
    }
    VC_TR(18);
    line_finish(s, cx, invfact, tr, b == 0, tid);
    __syncthreads();
    VC_TR(19);
}

}  // namespace vc
