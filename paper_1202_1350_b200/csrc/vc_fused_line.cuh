// vc_fused_line.cuh — step a7 inside the fused kernel: the line restriction q(t) = V~_{i+1}(l(t)), t = 2..s,
// l(t) = r1 + t (r2 - r1)  (reading c-5; absent from PAPER.md, which defers to [8],[10] at PAPER.md:85).
//
// One pass over V_{i+1}, organised as the binary fold tree of the multilinear extension with POLYNOMIALS IN t at the
// nodes: folding variable k of the table with l(t)_k raises the degree by one, so a node at level k is a polynomial of
// degree k.  A thread folds its 8 consecutive words over variables 0..2 (a cubic, built at t = 0..3 with 8 + 6 + 4 = 18
// multiplies; the extra node of each lower level comes from its finite differences) and continues it to P = tb + 4
// nodes t = 0..P-1 with three additions per node.  The block of 2^tb threads then folds variables 3..3+tb-1 in shared
// memory, one multiply per (node, t): about P multiplies per thread in all, instead of (s-1) multiply + warp-reduce
// steps.  The block's polynomial (degree <= P-1, known at P nodes) is continued to t = P..s by Lagrange interpolation on
// the integer nodes (integer coefficients from Pascal's triangle, 16 lanes per t), weighted with eq(block bits, l(t))
// and accumulated.
#pragma once
#include "vc_fused.cuh"

namespace vc {

__host__ __device__ inline uint32_t fused_line_tb(uint32_t s, uint32_t nthr) {
    const uint32_t sp = s < 3 ? 3 : s;
    uint32_t lg = 0;
    while ((2u << lg) <= nthr) lg++;
    return (sp - 3) < lg ? (sp - 3) : lg;
}
// grid-wide layers: blocks of 2^tb threads with tb chosen so that there are at least ~128 blocks to spread over the CTAs
__host__ __device__ inline uint32_t fused_line_tb_grid(uint32_t s, uint32_t nthr) {
    const uint32_t sp = s < 3 ? 3 : s, cap = sp > 10 ? sp - 10 : 0, tb = fused_line_tb(s, nthr);
    return tb < cap ? tb : cap;
}
// scratch words: pts[(s+1)*sp (even)] | A[2^tb * P] | B[2^tb * P / 2] | fx[32] | dl[32]
__host__ __device__ inline size_t fused_line_words(uint32_t s, uint32_t nthr) {
    const size_t sp = s < 3 ? 3 : s, tb = fused_line_tb(s, nthr), P = tb + 4, NB = (size_t)1 << tb;
    return (((s + 1) * sp + 1) & ~(size_t)1) + NB * P + (NB * P + 1) / 2 + 1 + 64;
}

// pas[n*32 + k] = C(n,k), n,k < 32 (C(31,15) < 2^32); threads tid < 32 fill one row each
__device__ __forceinline__ void build_pascal(uint32_t *pas, uint32_t tid) {
    if (tid < 32) {
        uint64_t c = 1;
        for (uint32_t k = 0; k < 32; k++) {
            pas[tid * 32 + k] = k <= tid ? (uint32_t)c : 0u;
            if (k < tid) c = c * (tid - k) / (k + 1);
        }
    }
}

// cx.acc[t-2] <- sum over this CTA's share (blocks vb0, vb0+vbstride, ...) of eq(u, l(t)) V[u], t = 2..s.
// Threads tid < nthr take part (nthr a power of two >= 32); they synchronise with bar_n(nthr).  Requires s >= 2.
__device__ __noinline__ void line_partials(const uint64_t *Vb, uint32_t s, FusedCtx &cx, const uint32_t *pas,
                                              uint64_t *scratch, uint32_t vb0, uint32_t vbstride, uint32_t tid, uint32_t nthr,
                                              uint32_t tb) {
    const uint32_t m = s - 1, sp = s < 3 ? 3 : s;
    const uint32_t P = tb + 4, NB = 1u << tb;
    const uint32_t nvb = 1u << (sp - 3 - tb);
    uint64_t *pts = scratch;                                     // pts[t*sp + k] = l(t)_k, t = 0..s; padded variables sit at 0
    uint64_t *A = pts + ((((size_t)s + 1) * sp + 1) & ~(size_t)1);
    uint64_t *B = A + (size_t)NB * P;
    uint64_t *fx = B + (((size_t)NB * P + 1) / 2 + 1 & ~(size_t)1);
    VC_TRL(70);
    for (uint32_t i = tid; i < m; i += nthr) cx.acc[i] = 0;
    {   // lane k of every warp owns variable k (sp <= 30); warp w takes t = w, w + nw, ...: l(t + nw) = l(t) + nw d, no division
        const uint32_t lane = tid & 31, w = tid >> 5, nw = nthr >> 5;
        if (lane < sp) {
            const uint64_t p = lane < s ? cx.r1[lane] : 0, q = lane < s ? cx.r2[lane] : 0, d = fp61::sub(q, p);
            const uint64_t step = nw == 1 ? d : fp61::mul(nw, d);
            uint64_t v = w == 0 ? p : fp61::add(p, fp61::mul(w, d));
            for (uint32_t t = w; t <= s; t += nw) { pts[t * sp + lane] = v; v = fp61::add(v, step); }
        }
    }
    // l(t)_k for k < 3 at t = 0..3
    uint64_t x[3][4];
#pragma unroll
    for (int k = 0; k < 3; k++) {
        const uint64_t p = (uint32_t)k < s ? cx.r1[k] : 0, q = (uint32_t)k < s ? cx.r2[k] : 0, d = fp61::sub(q, p);
        x[k][0] = p; x[k][1] = q; x[k][2] = fp61::add(q, d); x[k][3] = fp61::add(x[k][2], d);
    }
    VC_TRL(71);
    for (uint32_t vb = vb0; vb < nvb; vb += vbstride) {
        if (tid < NB) {
            uint64_t v[8];
            const size_t base = (((size_t)vb << tb) + tid) << 3;
            if (s >= 3) {
                const ulonglong2 *p2 = reinterpret_cast<const ulonglong2 *>(Vb + base);
#pragma unroll
                for (int e = 0; e < 4; e++) { const ulonglong2 w = p2[e]; v[2 * e] = w.x; v[2 * e + 1] = w.y; }
            } else {
#pragma unroll
                for (int e = 0; e < 8; e++) v[e] = base + e < ((size_t)1 << s) ? Vb[base + e] : 0;
            }
            // level 1: four linear polynomials at t = 0,1 (+ extrapolated t = 2)
            uint64_t f1[4][3];
#pragma unroll
            for (int e = 0; e < 4; e++) {
                const uint64_t d = fp61::sub(v[2 * e + 1], v[2 * e]);
                f1[e][0] = fp61::add(v[2 * e], fp61::mul(x[0][0], d));
                f1[e][1] = fp61::add(v[2 * e], fp61::mul(x[0][1], d));
                f1[e][2] = fp61::sub(fp61::dbl(f1[e][1]), f1[e][0]);
            }
            // level 2: two quadratics at t = 0,1,2 (+ extrapolated t = 3: f(3) = 3 f(2) - 3 f(1) + f(0))
            uint64_t f2[2][4];
#pragma unroll
            for (int e = 0; e < 2; e++) {
#pragma unroll
                for (int t = 0; t < 3; t++)
                    f2[e][t] = fp61::add(f1[2 * e][t], fp61::mul(x[1][t], fp61::sub(f1[2 * e + 1][t], f1[2 * e][t])));
                const uint64_t d21 = fp61::sub(f2[e][2], f2[e][1]);
                f2[e][3] = fp61::add(fp61::add(fp61::dbl(d21), d21), f2[e][0]);
            }
            // level 3: one cubic at t = 0..3, continued to t = 4..P-1 by its backward differences
            uint64_t f[4];
#pragma unroll
            for (int t = 0; t < 4; t++) {
                f[t] = fp61::add(f2[0][t], fp61::mul(x[2][t], fp61::sub(f2[1][t], f2[0][t])));
                A[(size_t)t * NB + tid] = f[t];
            }
            uint64_t cur = f[3];
            uint64_t d1 = fp61::sub(f[3], f[2]);
            uint64_t d2 = fp61::sub(d1, fp61::sub(f[2], f[1]));
            const uint64_t d3 = fp61::sub(d2, fp61::sub(fp61::sub(f[2], f[1]), fp61::sub(f[1], f[0])));
            for (uint32_t t = 4; t < P; t++) {
                d2 = fp61::add(d2, d3); d1 = fp61::add(d1, d2); cur = fp61::add(cur, d1);
                A[(size_t)t * NB + tid] = cur;
            }
        }
        VC_TRL(72);
        bar_n(nthr);                                             // also publishes pts on the first pass
        VC_TRL(73);
        // the block's fold tree over variables 3..3+tb-1: level lev halves the nodes, one multiply per (node, t)
        uint64_t *in = A, *out = B;
        for (uint32_t lev = 0; lev < tb; lev++) {
            const uint32_t lnout = tb - lev - 1, nout = 1u << lnout, var = 3 + lev;
            for (uint32_t item = tid; item < (P << lnout); item += nthr) {
                const uint32_t pt = item >> lnout, node = item & (nout - 1);
                const ulonglong2 ab = *reinterpret_cast<const ulonglong2 *>(in + ((size_t)pt << (lnout + 1)) + 2 * node);
                out[((size_t)pt << lnout) + node] = fold2(ab.x, ab.y, pts[pt * sp + var]);
            }
            bar_n(nthr);
            uint64_t *tmp = in; in = out; out = tmp;
        }
        VC_TRL(74);
        // in[pt], pt < P: the block polynomial.  Continue it to t = P..s.
        if (s + 1 > P) {
            // Lagrange on the integer nodes 0..P-1 at an integer t >= P:  f(t) = sum_i (-1)^(P-1-i) C(t,i) C(t-1-i, P-1-i) f(i)
            // (prod_{m != i}(t - m) / prod_{m != i}(i - m), an integer below 2^54 for t <= 30).  Sixteen lanes per t (P <= 13),
            // one multiply per lane, four shuffle steps: no serial pass over the nodes.
            if (tid < P) fx[tid] = in[tid];
            const uint32_t nit = (s + 1 - P) * 16;
            for (uint32_t base = 0; base < nit; base += nthr) {
                const uint32_t item = base + tid, t = P + (item >> 4), i = item & 15;
                uint64_t term = 0;
                if (item < nit && i < P) {
                    const uint64_t coef = (uint64_t)pas[t * 32 + i] * pas[(t - 1 - i) * 32 + (P - 1 - i)];
                    term = fp61::mul(coef, in[i]);
                    if ((P - 1 - i) & 1u) term = fp61::neg(term);
                }
#pragma unroll
                for (int off = 8; off; off >>= 1) term = fp61::add(term, __shfl_xor_sync(0xffffffffu, term, off));
                if (item < nit && i == 0) fx[t] = term;
            }
        } else if (tid <= s) {
            fx[tid] = in[tid];
        }
        bar_n(nthr);
        VC_TRL(75);
        if (tid >= 2 && tid <= s) {
            const uint64_t e = eq_direct(vb, pts + (size_t)tid * sp, 3 + tb, sp);     // eq(block bits, l(t))
            cx.acc[tid - 2] = fp61::add(cx.acc[tid - 2], fp61::mul(fx[tid], e));
        }
        VC_TRL(76);
        bar_n(nthr);
    }
    if (vb0 >= nvb) bar_n(nthr);                                 // pts / acc settled even without a block
}

// After the totals q[2..s] sit in cx.acc[0..s-1): warp 0 writes q[0..s] (if writer), draws tau, sets z <- l(tau),
// claim <- q(tau) by Lagrange interpolation on nodes 0..s, ctr += 1.  s <= 30.  The caller synchronises afterwards.
__device__ __noinline__ void line_finish(uint32_t s, FusedCtx &cx, const uint64_t *invfact, uint64_t *tr_q, bool writer,
                                            uint32_t tid) {
    if (tid >= 32) return;
    const uint32_t k = tid;
    const uint64_t tau = fp61::draw(cx.seed, cx.ctr);
    // prod_{mm != k} (tau - mm) for every lane k at once: prefix and suffix products of the factors across the warp
    // (five shuffle + multiply steps each, interleaved), instead of one serial pass over the nodes per lane
    const uint64_t f = k <= s ? fp61::sub(tau, k) : 1;
    uint64_t pre = f, suf = f;
#pragma unroll
    for (uint32_t off = 1; off < 32; off <<= 1) {
        const uint64_t up = __shfl_up_sync(0xffffffffu, pre, off), dn = __shfl_down_sync(0xffffffffu, suf, off);
        if (k >= off) pre = fp61::mul(pre, up);
        if (k + off < 32) suf = fp61::mul(suf, dn);
    }
    const uint64_t pl = __shfl_up_sync(0xffffffffu, pre, 1), sr = __shfl_down_sync(0xffffffffu, suf, 1);
    uint64_t term = 0;
    if (k <= s) {
        const uint64_t qk = k == 0 ? cx.v1 : (k == 1 ? cx.v2 : cx.acc[k - 2]);
        if (writer) tr_q[k] = qk;
        const uint64_t num = fp61::mul(k ? pl : 1, k < 31 ? sr : 1);
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
