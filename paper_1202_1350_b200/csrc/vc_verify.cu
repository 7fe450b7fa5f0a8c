// vc_verify.cu — vc_verify_transcript: the verifier of include/vc.h, host code (§2.2:
// V checks P's responses for internal consistency; the last claim is about an encoding of the
// input that V computes herself).  Not on the hot path (NEXT-1 in SURVEY.md §8(f) moves the two O(S) sums
// to the GPU).  Written independently of oracle/: Mersenne folding, closed-form degree-2 interpolation,
// factorial-table Lagrange weights.
#include <cstring>
#include <vector>

#include "fp61.cuh"
#include "vc_circuit.hpp"

namespace {

using u64 = uint64_t;

void eq_table(const u64 *x, uint32_t s, std::vector<u64> &T) {
    T.assign((size_t)1 << s, 0);
    T[0] = 1;
    for (uint32_t k = 0; k < s; k++) {
        const size_t half = (size_t)1 << k;
        for (size_t u = 0; u < half; u++) {
            const u64 hi = fp61::mul(T[u], x[k]);
            T[u + half] = hi;
            T[u] = fp61::sub(T[u], hi);
        }
    }
}

u64 mle(const u64 *V, uint32_t s, const u64 *x) {
    // fold one variable at a time, LSB first
    std::vector<u64> A(V, V + ((size_t)1 << s));
    for (uint32_t k = 0; k < s; k++) {
        const size_t half = (size_t)1 << (s - k - 1);
        for (size_t u = 0; u < half; u++) A[u] = fp61::add(A[2 * u], fp61::mul(x[k], fp61::sub(A[2 * u + 1], A[2 * u])));
    }
    return A[0];
}

// g(r) for the quadratic through (0,G0),(1,G1),(2,G2):  G0 (r-1)(r-2)/2 - G1 r (r-2) + G2 r (r-1)/2
u64 interp2(const u64 *G, u64 r) {
    const u64 half = 1ull << 60;  // 1/2 mod p
    const u64 rm1 = fp61::sub(r, 1), rm2 = fp61::sub(r, 2);
    const u64 l0 = fp61::mul(fp61::mul(rm1, rm2), half);
    const u64 l1 = fp61::neg(fp61::mul(r, rm2));
    const u64 l2 = fp61::mul(fp61::mul(r, rm1), half);
    return fp61::add(fp61::add(fp61::mul(G[0], l0), fp61::mul(G[1], l1)), fp61::mul(G[2], l2));
}

u64 fpow(u64 a, u64 e) {
    u64 r = 1;
    while (e) { if (e & 1) r = fp61::mul(r, a); a = fp61::mul(a, a); e >>= 1; }
    return r;
}

// q(tau) for the polynomial of degree <= s with q[k] at node k
u64 lagrange(const u64 *q, uint32_t s, u64 tau) {
    std::vector<u64> pre(s + 2, 1), suf(s + 2, 1), invf(s + 1);
    for (uint32_t k = 0; k <= s; k++) pre[k + 1] = fp61::mul(pre[k], fp61::sub(tau, k));
    for (int k = (int)s; k >= 0; k--) suf[k] = fp61::mul(suf[k + 1], fp61::sub(tau, (u64)k));
    u64 f = 1;
    for (uint32_t k = 1; k <= s; k++) f = fp61::mul(f, k);
    u64 inv = fpow(f, fp61::P - 2);
    for (int k = (int)s; k >= 0; k--) { invf[k] = inv; inv = fp61::mul(inv, (u64)k); }
    u64 tot = 0;
    for (uint32_t k = 0; k <= s; k++) {
        u64 term = fp61::mul(fp61::mul(q[k], fp61::mul(pre[k], suf[k + 1])), fp61::mul(invf[k], invf[s - k]));
        if ((s - k) & 1) term = fp61::neg(term);
        tot = fp61::add(tot, term);
    }
    return tot;
}

u64 gate_fn(uint32_t t, u64 L, u64 R) {
    switch (t) {
    case VC_ADD: return fp61::add(L, R);
    case VC_MULT: return fp61::mul(L, R);
    case VC_SUB: return fp61::sub(L, R);
    default: return L;
    }
}

}  // namespace

extern "C" int vc_verify_transcript(const vc_circuit *c, const uint64_t *h_input, const uint64_t *h_outputs, uint64_t seed,
                                    const uint64_t *h_transcript, uint64_t n_words, int *accept, uint32_t *fail_layer,
                                    uint32_t *fail_round) {
    if (!c || !h_input || !h_outputs || !h_transcript || !accept || !fail_layer || !fail_round) return VC_ERR_ARG;
    *accept = 0; *fail_layer = 0; *fail_round = 0;
    if (n_words != c->total_words) return VC_ERR_ARG;
    for (size_t u = 0; u < ((size_t)1 << c->log_input); u++) if (h_input[u] >= fp61::P) return VC_ERR_ARG;
    for (size_t u = 0; u < ((size_t)1 << c->logs[0]); u++) if (h_outputs[u] >= fp61::P) return VC_ERR_ARG;
    for (uint64_t w = 0; w < n_words; w++) if (h_transcript[w] >= fp61::P) return VC_ERR_ARG;
    try {
        u64 z[vc::MAX_VARS], r[2 * vc::MAX_VARS], ctr = 0, claim;
        for (uint32_t k = 0; k < c->logs[0]; k++) z[k] = fp61::draw(seed, ctr++);
        claim = mle(h_outputs, c->logs[0], z);
        const u64 *tr = h_transcript;
        std::vector<u64> Tz, T1, T2;
        for (uint32_t i = 0; i < c->d; i++) {
            const uint32_t s = c->logs[i + 1];
            if (i == 0 && c->sum_out) {          // the sum gate (VC_SUM in vc.h): s linear rounds, then the claim is V~_1(r) at z = r
                for (uint32_t m = 0; m < s; m++, tr += 2) {
                    if (fp61::add(tr[0], tr[1]) != claim) { *fail_layer = 0; *fail_round = m; return VC_OK; }
                    z[m] = fp61::draw(seed, ctr++);
                    claim = fp61::add(tr[0], fp61::mul(z[m], fp61::sub(tr[1], tr[0])));
                }
                continue;
            }
            for (uint32_t m = 0; m < 2 * s; m++, tr += 3) {
                if (fp61::add(tr[0], tr[1]) != claim) { *fail_layer = i; *fail_round = m; return VC_OK; }
                r[m] = fp61::draw(seed, ctr++);
                claim = interp2(tr, r[m]);
            }
            const u64 *q = tr; tr += s + 1;
            eq_table(z, c->logs[i], Tz); eq_table(r, s, T1); eq_table(r + s, s, T2);
            u64 W[4] = {0, 0, 0, 0};
            const auto &ty = c->h_type[i]; const auto &a = c->h_in1[i]; const auto &b = c->h_in2[i];
            for (size_t g = 0; g < ty.size(); g++)
                W[ty[g]] = fp61::add(W[ty[g]], fp61::mul(Tz[g], fp61::mul(T1[a[g]], T2[b[g]])));
            u64 rhs = 0;
            for (uint32_t t = 0; t < 4; t++) rhs = fp61::add(rhs, fp61::mul(W[t], gate_fn(t, q[0], q[1])));
            if (rhs != claim) { *fail_layer = i; *fail_round = 2 * s; return VC_OK; }
            const u64 tau = fp61::draw(seed, ctr++);
            for (uint32_t k = 0; k < s; k++) z[k] = fp61::add(r[k], fp61::mul(tau, fp61::sub(r[s + k], r[k])));
            claim = lagrange(q, s, tau);
        }
        if (mle(h_input, c->log_input, z) != claim) { *fail_layer = c->d; *fail_round = 0; return VC_OK; }
    } catch (const std::bad_alloc &) { return VC_ERR_NOMEM; }
    *accept = 1;
    return VC_OK;
}
