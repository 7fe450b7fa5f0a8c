// vc_fused_small.cuh — one narrow layer (<= 2^10 gates, table <= 2^12 words) proved by a single CTA out of shared
// memory: one gate per thread in registers, fold tables in shared memory, block barriers only (steps a2-a7).
#pragma once
#include "vc_fused.cuh"

namespace vc {

__device__ __forceinline__ void small_layer(const FusedArgs &a, FusedCtx &cx, uint8_t *dyn, uint32_t layer, uint64_t *tr) {
    const uint32_t tid = threadIdx.x;
    const LayerDesc Li = a.L[layer], Lb = a.L[layer + 1];
    const uint32_t si = Li.log_n, s = Lb.log_n;
    const uint32_t n = 1u << si, nb = 1u << s;
    uint64_t *Vs = reinterpret_cast<uint64_t *>(dyn);           // V_{i+1}, 2^s words
    uint64_t *A0 = Vs + (1u << F_SMALL_T_LOG);                   // fold ping-pong: 2^(s-1), 2^(s-2)
    uint64_t *A1 = A0 + (1u << (F_SMALL_T_LOG - 1));
    uint64_t *E = A1 + (1u << (F_SMALL_T_LOG - 2));              // beta table, 2^si words
    uint64_t *scratch = E + (1u << F_SMALL_N_LOG);               // line restriction scratch
    for (uint32_t u = tid; u < nb; u += FT) Vs[u] = Lb.V[u];
    build_eq_low(E, cx.z, si);                                   // a3 (trailing barrier covers Vs too)
    const bool live = tid < n;
    uint64_t Pg = live ? E[tid] : 0;
    uint32_t i1 = 0, i2 = 0, t = 3;
    if (live) { i1 = Li.in1[tid]; i2 = Li.in2[tid]; t = Li.type[tid]; }
    const uint64_t w = Vs[i2];
    if (layer == 0) {                                            // a2
        uint64_t v[3] = {live ? fp61::mul(Pg, Li.V[tid]) : 0, 0, 0};
        block_reduce3(cx, v);
        if (tid == 0) cx.claim = cx.acc[0];
    }
    for (int phase = 1; phase <= 2; phase++) {
        const uint32_t idx = phase == 1 ? i1 : i2;
        const uint64_t *tab = Vs;
        for (uint32_t j = 0; j < s; j++) {
            acc128 a0, a1, a2; a0.clear(); a1.clear(); a2.clear();
            const uint32_t bit = (idx >> j) & 1u, u = idx >> (j + 1);
            const uint64_t lo = tab[2 * u], hi = tab[2 * u + 1];
            if (phase == 1) gate_terms<1>(t, Pg, w, bit, lo, hi, a0, a1, a2);
            else gate_terms<2>(t, Pg, cx.v1, bit, lo, hi, a0, a1, a2);
            uint64_t v3[3] = {a0.value(), a1.value(), a2.value()};
            block_reduce3(cx, v3);
            const uint64_t r = fp61::draw(cx.seed, cx.ctr);
            if (tid < 3) tr[tid] = cx.acc[tid];
            tr += 3;
            Pg = fp61::mul(Pg, bit ? r : fp61::sub(1, r));       // a6
            uint64_t *out = (j & 1) ? A1 : A0;
            const uint32_t half = nb >> (j + 1);
            for (uint32_t v = tid; v < half; v += FT) out[v] = fold2(tab[2 * v], tab[2 * v + 1], r);
            __syncthreads();
            if (tid == 0) { cx.ctr += 1; if (phase == 1) cx.r1[j] = r; else cx.r2[j] = r; }
            tab = out;
        }
        if (tid == 0) { if (phase == 1) cx.v1 = tab[0]; else cx.v2 = tab[0]; }
        __syncthreads();
    }
    if (s > 1) line_partials(Lb.V, s, cx, scratch, 0, 1);
    line_finish(s, cx, a.st, tr, true);
}

constexpr size_t F_SMALL_BYTES = ((1u << F_SMALL_T_LOG) + (1u << (F_SMALL_T_LOG - 1)) + (1u << (F_SMALL_T_LOG - 2)) +
                                  (1u << F_SMALL_N_LOG)) * 8 + (64 * 64 + 3 * 64 * 32) * 8;
static_assert(F_SMALL_BYTES <= F_STATE_BYTES, "small-layer buffers alias the gate-state region");

}  // namespace vc
