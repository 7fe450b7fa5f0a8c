// vc_fused_line.cuh — step a7 inside the fused kernel: the line restriction q(t) = V~_{i+1}(l(t)), t = 2..s,
// l(t) = r1 + t (r2 - r1)  (reading c-5; absent from PAPER.md, which defers to [8],[10] at PAPER.md:85).
//
// One pass over V_{i+1}.  A thread holds 8 consecutive words.  Folding them over the first three variables gives a
// polynomial of degree 3 in t; it is built at t = 0..3 with 8 + 6 + 4 = 18 multiplies (level k has degree k, the
// extra node of the lower level comes from its finite differences), and then continued to t = 4..s with three
// additions per node (backward differences of a cubic).  Each node is weighted by eq(rest of the index, l(t)):
// lane bits and warp bits from two small tables, block bits by one product per (block, t).
#pragma once
#include "vc_fused.cuh"

namespace vc {

// scratch words needed: m*sp + 3*m*32 with m = s-1, sp = max(s,3)
__host__ __device__ inline size_t fused_line_words(uint32_t s) {
    const size_t m = s > 1 ? s - 1 : 0, sp = s < 3 ? 3 : s;
    return m * sp + 3 * m * 32;
}

// cx.acc[t-2] <- sum over this CTA's share (blocks vb0, vb0+vbstride, ...) of eq(u, l(t)) V[u], t = 2..s.
// Threads tid < nthr take part (nthr a power of two >= 32); they synchronise with bar_n(nthr).  Requires s >= 2.
__device__ __forceinline__ void line_partials(const uint64_t *Vb, uint32_t s, FusedCtx &cx, uint64_t *scratch,
                                              uint32_t vb0, uint32_t vbstride, uint32_t tid, uint32_t nthr) {
    const uint32_t m = s - 1, sp = s < 3 ? 3 : s, lane = tid & 31, warp = tid >> 5;
    const uint32_t lg = 31 - __clz(nthr);
    const uint32_t tb = (sp - 3) < lg ? (sp - 3) : lg;        // index bits covered by the threads of one block
    const uint32_t lb = tb < 5 ? tb : 5, wb = tb - lb;
    const uint32_t nvb = 1u << (sp - 3 - tb);
    uint64_t *pts = scratch, *Wl = pts + (size_t)m * sp, *Ww = Wl + (size_t)m * 32, *red = Ww + (size_t)m * 32;
    for (uint32_t i = tid; i < m; i += nthr) cx.acc[i] = 0;
    for (uint32_t i = tid; i < m * sp; i += nthr) {
        const uint32_t t = i / sp + 2, k = i % sp;
        pts[i] = k < s ? fp61::add(cx.r1[k], fp61::mul(t, fp61::sub(cx.r2[k], cx.r1[k]))) : 0;   // padded variables sit at 0
    }
    bar_n(nthr);
    for (uint32_t i = tid; i < m * 32; i += nthr) {
        const uint32_t t = i >> 5, l = i & 31;
        uint64_t e = 1, f = 1;
        for (uint32_t k = 0; k < lb; k++) e = fp61::mul(e, fp61::chi((l >> k) & 1u, pts[t * sp + 3 + k]));
        for (uint32_t k = 0; k < wb; k++) f = fp61::mul(f, fp61::chi((l >> k) & 1u, pts[t * sp + 3 + lb + k]));
        Wl[i] = (l < (1u << lb)) ? e : 0;
        Ww[i] = (l < (1u << wb)) ? f : 0;
    }
    // l(t)_k for k < 3 at t = 0..3
    uint64_t x[3][4];
#pragma unroll
    for (int k = 0; k < 3; k++) {
        const uint64_t p = (uint32_t)k < s ? cx.r1[k] : 0, q = (uint32_t)k < s ? cx.r2[k] : 0, d = fp61::sub(q, p);
        x[k][0] = p; x[k][1] = q; x[k][2] = fp61::add(q, d); x[k][3] = fp61::add(x[k][2], d);
    }
    const bool active = tid < (1u << tb);
    const uint32_t nwu = (1u << tb) > 32 ? (1u << tb) >> 5 : 1;
    for (uint32_t vb = vb0; vb < nvb; vb += vbstride) {
        bar_n(nthr);                                           // tables ready / red free again
        if (warp < nwu) {
            uint64_t v[8];
            const size_t base = (((size_t)vb << tb) + tid) << 3;
#pragma unroll
            for (int e = 0; e < 8; e++) v[e] = (active && base + e < ((size_t)1 << s)) ? Vb[base + e] : 0;
            // level 1: four linear polynomials at t = 0,1
            uint64_t f1[4][3];
#pragma unroll
            for (int e = 0; e < 4; e++) {
                const uint64_t d = fp61::sub(v[2 * e + 1], v[2 * e]);
                f1[e][0] = fp61::add(v[2 * e], fp61::mul(x[0][0], d));
                f1[e][1] = fp61::add(v[2 * e], fp61::mul(x[0][1], d));
                f1[e][2] = fp61::sub(fp61::dbl(f1[e][1]), f1[e][0]);                 // extrapolated node t = 2
            }
            // level 2: two quadratics at t = 0,1,2, extended to t = 3
            uint64_t f2[2][4];
#pragma unroll
            for (int e = 0; e < 2; e++) {
#pragma unroll
                for (int t = 0; t < 3; t++)
                    f2[e][t] = fp61::add(f1[2 * e][t], fp61::mul(x[1][t], fp61::sub(f1[2 * e + 1][t], f1[2 * e][t])));
                // f(3) = 3 f(2) - 3 f(1) + f(0)
                const uint64_t d21 = fp61::sub(f2[e][2], f2[e][1]);
                f2[e][3] = fp61::add(fp61::add(fp61::dbl(d21), d21), f2[e][0]);
            }
            // level 3: one cubic at t = 0..3
            uint64_t f[4];
#pragma unroll
            for (int t = 0; t < 4; t++) f[t] = fp61::add(f2[0][t], fp61::mul(x[2][t], fp61::sub(f2[1][t], f2[0][t])));
            // backward differences at t = 3
            uint64_t cur = f[2];
            uint64_t d1 = fp61::sub(f[3], f[2]);
            uint64_t d2 = fp61::sub(d1, fp61::sub(f[2], f[1]));
            const uint64_t d3 = fp61::sub(d2, fp61::sub(fp61::sub(f[2], f[1]), fp61::sub(f[1], f[0])));
            for (uint32_t ti = 0; ti < m; ti++) {              // node t = ti + 2
                if (ti == 1) cur = f[3];
                else if (ti >= 2) { d2 = fp61::add(d2, d3); d1 = fp61::add(d1, d2); cur = fp61::add(cur, d1); }
                uint64_t val = active ? fp61::mul(cur, Wl[ti * 32 + lane]) : 0;
                val = warp_sum61(val);
                if (lane == 0) red[ti * 32 + warp] = fp61::mul(val, Ww[ti * 32 + warp]);
            }
        }
        bar_n(nthr);
        for (uint32_t ti = tid; ti < m; ti += nthr) {
            uint64_t sum = 0;
            for (uint32_t w = 0; w < nwu; w++) sum = fp61::add(sum, red[ti * 32 + w]);
            uint64_t e = 1;
            for (uint32_t k = 3 + tb; k < sp; k++) e = fp61::mul(e, fp61::chi((vb >> (k - 3 - tb)) & 1u, pts[ti * sp + k]));
            cx.acc[ti] = fp61::add(cx.acc[ti], fp61::mul(sum, e));
        }
    }
    bar_n(nthr);
}

// After the totals q[2..s] sit in cx.acc[0..s-1): warp 0 writes q[0..s] (if writer), draws tau, sets z <- l(tau),
// claim <- q(tau) by Lagrange interpolation on nodes 0..s, ctr += 1.  s <= 30.  The caller synchronises afterwards.
__device__ __forceinline__ void line_finish(uint32_t s, FusedCtx &cx, const uint64_t *invfact, uint64_t *tr_q, bool writer,
                                            uint32_t tid) {
    if (tid >= 32) return;
    const uint32_t k = tid;
    const uint64_t tau = fp61::draw(cx.seed, cx.ctr);
    uint64_t term = 0;
    if (k <= s) {
        const uint64_t qk = k == 0 ? cx.v1 : (k == 1 ? cx.v2 : cx.acc[k - 2]);
        if (writer) tr_q[k] = qk;
        uint64_t c[4] = {1, 1, 1, 1};                          // prod_{mm != k} (tau - mm), four interleaved chains
        for (uint32_t mm = 0; mm <= s; mm += 4) {
#pragma unroll
            for (uint32_t e = 0; e < 4; e++)
                if (mm + e <= s && mm + e != k) c[e] = fp61::mul(c[e], fp61::sub(tau, mm + e));
        }
        const uint64_t num = fp61::mul(fp61::mul(c[0], c[1]), fp61::mul(c[2], c[3]));
        const uint64_t dinv = fp61::mul(invfact[k], invfact[s - k]);
        term = fp61::mul(qk, fp61::mul(num, dinv));
        if ((s - k) & 1u) term = fp61::neg(term);
    }
    const uint64_t claim = warp_sum61(term);
    uint64_t znew = 0;
    if (k < s) znew = fold2(cx.r1[k], cx.r2[k], tau);
    __syncwarp();
    if (k < s) cx.z[k] = znew;
    if (k == 0) { cx.claim = claim; cx.ctr += 1; }
}

}  // namespace vc
