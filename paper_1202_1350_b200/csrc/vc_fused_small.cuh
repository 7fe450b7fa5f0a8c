// vc_fused_small.cuh — one narrow layer (<= 2^8 gates: F_SMALL_N_LOG, table <= 2^12 words) proved by a single CTA out of shared
// memory (steps a2-a7).  One gate per thread in registers; only as many warps as the layer needs take part and they
// synchronise on a named barrier, so a round of a 1-gate layer costs two 1-warp barriers, not two 32-warp ones.
// Per round: contributions -> 3 warp REDUX sums -> barrier (message complete) -> challenge -> weight update and
// table fold -> barrier.  Warp 0 sums the per-warp partials and writes the transcript off the critical path.
#pragma once
#include "vc_fused.cuh"
#include "vc_fused_line.cuh"

namespace vc {

constexpr size_t F_SMALL_WORDS = (1u << F_SMALL_T_LOG) + (1u << (F_SMALL_T_LOG - 1)) + (1u << (F_SMALL_T_LOG - 2)) + 2 * 32 * 4;

// per-type (W, c, ignore-x) of a gate for a phase:  contribution = W * (x + c)   (x := 0 when ignore)
//   phase 1 (x = V~(w1) side, other = V[in2]):  MULT (P*other, 0)  ADD (P, other)  SUB (P, -other)  RELAY (P, 0)
//   phase 2 (x = V~(w2) side, other = v1):      MULT (P*v1, 0)     ADD (P, v1)     SUB (-P, -v1)    RELAY (P, v1; x ignored)
__device__ __forceinline__ void gate_state(int phase, uint32_t t, uint64_t P, uint64_t other, uint64_t &W, uint64_t &c,
                                           uint32_t &ign) {
    ign = 0;
    if (t == VC_MULT) { W = fp61::mul(P, other); c = 0; }
    else if (t == VC_ADD) { W = P; c = other; }
    else if (t == VC_SUB) { W = phase == 1 ? P : fp61::neg(P); c = fp61::neg(other); }
    else { W = P; c = phase == 1 ? 0 : other; ign = phase == 1 ? 0u : 1u; }
}

__device__ __forceinline__ void small_layer(const FusedArgs &a, FusedCtx &cx, const uint64_t *invfact, const uint32_t *pas, uint8_t *dyn,
                                            uint32_t layer, uint64_t *tr) {
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t si = a.L[layer].log_n, s = a.L[layer + 1].log_n;
    const uint32_t n = 1u << si, nb = 1u << s;                   // n <= 2^F_SMALL_N_LOG <= 256, nb <= 2^F_SMALL_T_LOG
    uint64_t *Vs = reinterpret_cast<uint64_t *>(dyn);            // level 0: V_{i+1}
    uint64_t *X = Vs + (1u << F_SMALL_T_LOG);                     // odd levels
    uint64_t *Y = X + (1u << (F_SMALL_T_LOG - 1));                // even levels >= 2
    ulonglong2 *cbuf = reinterpret_cast<ulonglong2 *>(Y + (1u << (F_SMALL_T_LOG - 2)));   // [2][256] committed products
    uint64_t *sred = reinterpret_cast<uint64_t *>(cbuf + 2 * 256);
    uint64_t *scratch = sred + 32;
    __syncthreads();                                             // bookkeeping of the previous layer is settled
    const uint64_t *Vg = a.L[layer + 1].V;
    for (uint32_t u = tid; u < nb; u += FT) Vs[u] = __ldcg(Vg + u);
    const bool live = tid < n;
    uint64_t P = live ? eq_direct(tid, cx.z, 0, si) : 0;         // a3: beta(z, g) by direct product
    uint32_t i1 = 0, i2 = 0, t = VC_RELAY;
    if (live) Wires(a.L[layer], &cx.wrule).get(tid, i1, i2, t);
    uint32_t ctr = (uint32_t)cx.ctr;
    const uint64_t seed = cx.seed;
    __syncthreads();
    if (layer == 0) {                                            // a2: start claim V~_0(z_0) = sum_g beta(z_0,g) V_0[g]
        const uint64_t v = warp_sum61(live ? fp61::mul(P, a.L[0].V[tid]) : 0);
        if (lane == 0) sred[warp] = v;
        __syncthreads();
        if (warp == 0) {
            const uint64_t tot = warp_sum61(lane < (uint32_t)FT / 32 ? sred[lane] : 0);
            if (lane == 0) cx.claim = tot;
        }
        __syncthreads();
    }
    uint32_t par = 0;
    VC_TR(1);
    for (int phase = 1; phase <= 2; phase++) {
        const uint32_t idx = phase == 1 ? i1 : i2;
        uint64_t W = 0, c = 0; uint32_t ign = 0;
        if (live) gate_state(phase, t, P, phase == 1 ? Vs[i2] : cx.v1, W, c, ign);
        const uint64_t cP = c + fp61::P;
        for (uint32_t j = 0; j < s; j++) {
            const uint64_t *tab = j == 0 ? Vs : ((j & 1) ? X : Y);
            const uint32_t bit = (idx >> j) & 1u;
            if (live) {                                          // a4: this thread's gate; its two products are committed
                const uint32_t u = idx >> (j + 1);
                uint64_t lo = tab[2 * u], hi = tab[2 * u + 1];
                if (ign) { lo = 0; hi = 0; }
                const uint64_t mb = (bit ? hi : lo) + cP, m2 = 2 * hi + cP - lo;
                ulonglong2 o;
                o.x = fp61::fold128(fp61::mulhi(W, mb), W * mb) | ((uint64_t)bit << 63);
                o.y = fp61::fold128(fp61::mulhi(W, m2), W * m2);
                cbuf[par * 256 + tid] = o;
            }
            VC_TR(2);
            __syncthreads();                                     // every contribution to message j is committed
            VC_TR(3);
            if (warp == 15) {                                    // a5 off the critical path: G[0..2] -> transcript
                const ulonglong2 *cb = cbuf + par * 256;
                uint64_t X0l = 0, X1l = 0, Y0l = 0, Y1l = 0; uint32_t X0h = 0, X1h = 0, Y0h = 0, Y1h = 0;
                for (uint32_t i = lane; i < n; i += 32) {
                    const ulonglong2 q = cb[i];
                    const uint32_t b1 = (uint32_t)(q.x >> 63);
                    const uint64_t v1 = q.x & ~(1ull << 63);
                    add_c(X0l, X0h, v1, b1 ^ 1u); add_c(X1l, X1h, v1, b1);
                    add_c(Y0l, Y0h, q.y, b1 ^ 1u); add_c(Y1l, Y1h, q.y, b1);
                }
                const uint64_t t0 = warp_sum61(fp61::fold128(X0h, X0l)), t1 = warp_sum61(fp61::fold128(X1h, X1l));
                const uint64_t y0 = fp61::fold128(Y0h, Y0l), y1 = fp61::fold128(Y1h, Y1l);
                const uint64_t t2 = warp_sum61(fp61::sub(fp61::dbl(y1), y0));
                if (lane < 3) tr[lane] = lane == 0 ? t0 : (lane == 1 ? t1 : t2);
            } else {                                             // a6: challenge, weight update, fold
                const uint32_t half = nb >> (j + 1);
                if (tid < n || tid < half) {                     // idle warps go straight to the barrier
                    const uint64_t r = fp61::draw(seed, ctr);
                    if (live) {
                        const uint64_t f = bit ? r : fp61::sub(1, r);
                        W = fp61::mul(W, f); P = fp61::mul(P, f);
                    }
                    uint64_t *out = ((j + 1) & 1) ? X : Y;
                    for (uint32_t v = tid; v < half; v += F_WORKERS) out[v] = fold2(tab[2 * v], tab[2 * v + 1], r);
                    if (tid == 0) { if (phase == 1) cx.r1[j] = r; else cx.r2[j] = r; }
                }
                VC_TR(4);
                bar_workers();
                VC_TR(5);
            }
            ctr++; tr += 3; par ^= 1;
        }
        __syncthreads();                                         // the reducer is done; level s and r[] are visible to all
        const uint64_t vend = ((s & 1) ? X : Y)[0];               // level s: V~_{i+1}(r1) resp. (r2)
        if (tid == 0) { if (phase == 1) cx.v1 = vend; else cx.v2 = vend; }
        // P now equals beta(z,g) eq(in1[g], r1): the plain weight phase 2 starts from
        __syncthreads();
    }
    if (tid == 0) cx.ctr = ctr;
    VC_TR(6);
    uint32_t nthr = 32;
    while (nthr < (nb >> 3) && nthr < (uint32_t)FT) nthr <<= 1;   // the line restriction wants 2^(s-3) threads
    __syncthreads();
    if (tid < nthr && s > 1) line_partials(Vs, s, cx, pas, scratch, 0, 1, tid, nthr, fused_line_tb(s, nthr));   // a7
    __syncthreads();
    VC_TR(7);
    line_finish(s, cx, invfact, tr, true, tid);
    VC_TR(8);
    __syncthreads();
}

constexpr size_t F_SMALL_BYTES = (F_SMALL_WORDS + 2 * 256 * 2 + 32 + 13 * 12 + 2 + 512 * 13 + 256 * 13 + 2 + 64) * 8;   // + commit + line scratch, s <= 12

}  // namespace vc
