// vc_verify_gpu.cu — vc_verify_transcript_device: the verifier with its O(S) sums on the GPU.
//
// PAPER.md:127 (§4.1.2): the verifier's own work is dominated by evaluating the low-degree extension of the input at
// one random point — every input element contributes one chi-weighted term, terms are summed in F_p ("each thread
// computes the contribution of one input element, followed by a parallel reduction"); this is where the
// paper's > 100x client speedup comes from.  In the GKR form used here (readings c-2, c-5) the verifier has
// three kinds of O(S) sums, all of the same shape (a product of eq factors per element, reduced mod p):
//     start claim    V~_0(z_0)        = sum_g eq(g, z_0) V_0[g]                         (claimed outputs)
//     wiring sums    W_t(z, r1, r2)   = sum_{g of type t} eq(g,z) eq(in1[g],r1) eq(in2[g],r2)   per layer, t = 0..3
//     closing check  V~_d(z_d)        = sum_u eq(u, z_d) x[u]                           (the input: V's "secret")
// Every point (z_i, r1_i, r2_i) is a function of the seed alone (the challenges do not depend on the messages,
// reading c-18), so all d + 2 kernels are enqueued at once; the O(rounds) consistency checks then run on the host
// over the 7s+1 transcript words per layer, exactly as in vc_verify.cu, with the device sums plugged in.
// Nothing here is shared with oracle/, nor with the prover's kernels beyond fp61.cuh.
#include <algorithm>
#include <new>
#include <cstring>
#include <vector>

#include "fp61.cuh"
#include "vc_circuit.hpp"

namespace vc {

using fp61::acc128;
constexpr int VT = 512;                                   // threads per block of the verifier kernels
constexpr uint32_t V_EQLOG = 10;                          // eq tables: 2^10 entries for variables 0..9, 2^10 for 10..19
constexpr size_t V_TAB_WORDS = (2u << V_EQLOG) + 128;     // one two-level eq table + the four 5-variable factors
constexpr int V_MAX_BLOCKS = 296;                         // 2 per SM: every block builds its own tables

__device__ __forceinline__ uint64_t warp_sum61(uint64_t v) {  // every lane gets the canonical total
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v = fp61::add(v, __shfl_xor_sync(0xffffffffu, v, d));
    return v;
}
// eq(u, x[k0..k1)) = prod_k chi(bit k-k0 of u, x[k]) by direct product
__device__ __forceinline__ uint64_t eq_prod(uint32_t u, const uint64_t *x, uint32_t k0, uint32_t k1) {
    uint64_t e = 1;
    for (uint32_t k = k0; k < k1; k++) e = fp61::mul(e, fp61::chi((u >> (k - k0)) & 1u, x[k]));
    return e;
}
// two-level eq table over nv variables: lo[u] = eq(u, x[0..cl)), hi[w] = eq(w, x[cl..ch)); variables >= 20 per index
struct EqTab {
    const uint64_t *lo, *hi, *x;
    uint32_t nv;
    __device__ __forceinline__ uint64_t eq_of(uint32_t u) const {
        uint64_t e = lo[u & ((1u << V_EQLOG) - 1)];
        if (nv > V_EQLOG) e = fp61::mul(e, hi[(u >> V_EQLOG) & ((1u << V_EQLOG) - 1)]);
        if (nv > 2 * V_EQLOG) e = fp61::mul(e, eq_prod(u >> (2 * V_EQLOG), x, 2 * V_EQLOG, nv));
        return e;
    }
};
// All threads of the block (one block barrier inside); the caller synchronises afterwards.  Each 2^10-entry half is the
// outer product of two tables over at most 5 variables (built by direct product in tmp[0..128)): one multiply per entry.
__device__ __forceinline__ EqTab build_eq_tab(uint64_t *tab, uint64_t *tmp, const uint64_t *x, uint32_t nv, uint32_t tid) {
    const uint32_t cl = nv < V_EQLOG ? nv : V_EQLOG, ch = nv < 2 * V_EQLOG ? nv : 2 * V_EQLOG, hv = ch - cl;
    const uint32_t la = cl < 5 ? cl : 5, lb = cl - la, ha = hv < 5 ? hv : 5, hb = hv - ha;
    uint64_t *lo = tab, *hi = tab + (1u << V_EQLOG);
    if (tid < 128) {
        const uint32_t which = tid >> 5, u = tid & 31;
        if (which == 0) { if (u < (1u << la)) tmp[u] = eq_prod(u, x, 0, la); }
        else if (which == 1) { if (u < (1u << lb)) tmp[32 + u] = eq_prod(u, x, la, cl); }
        else if (which == 2) { if (u < (1u << ha)) tmp[64 + u] = eq_prod(u, x, cl, cl + ha); }
        else if (u < (1u << hb)) tmp[96 + u] = eq_prod(u, x, cl + ha, ch);
    }
    __syncthreads();
    for (uint32_t u = tid; u < (1u << cl); u += VT) lo[u] = fp61::mul(tmp[u & ((1u << la) - 1)], tmp[32 + (u >> la)]);
    for (uint32_t u = tid; u < (1u << hv); u += VT) hi[u] = fp61::mul(tmp[64 + (u & ((1u << ha) - 1))], tmp[96 + (u >> ha)]);
    EqTab e; e.lo = lo; e.hi = hi; e.x = x; e.nv = nv;
    return e;
}

// block partials -> part[block * K + k]; the block that takes the last ticket sums them into out[0..K)
template <int K>
__device__ __forceinline__ void verifier_reduce(uint64_t (&v)[K], uint64_t *red, uint64_t *part, unsigned *ticket, uint64_t *out) {
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    __shared__ unsigned s_last;
#pragma unroll
    for (int k = 0; k < K; k++) v[k] = warp_sum61(v[k]);
    __syncthreads();
    if (lane == 0) {
#pragma unroll
        for (int k = 0; k < K; k++) red[k * 32 + warp] = v[k];
    }
    __syncthreads();
    if (warp == 0) {
#pragma unroll
        for (int k = 0; k < K; k++) {
            const uint64_t t = warp_sum61(lane < VT / 32 ? red[k * 32 + lane] : 0);
            if (lane == 0) __stcg(part + (size_t)blockIdx.x * K + k, t);
        }
        if (lane == 0) { __threadfence(); s_last = atomicAdd(ticket, 1u) == gridDim.x - 1 ? 1u : 0u; }
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
#pragma unroll
    for (int k = 0; k < K; k++) {
        uint64_t a = 0;
        for (uint32_t b = tid; b < gridDim.x; b += VT) a = fp61::add(a, __ldcg(part + (size_t)b * K + k));
        a = warp_sum61(a);
        __syncthreads();
        if (lane == 0) red[warp] = a;
        __syncthreads();
        if (warp == 0) {
            const uint64_t t = warp_sum61(lane < VT / 32 ? red[lane] : 0);
            if (lane == 0) out[k] = t;
        }
    }
    if (tid == 0) *ticket = 0;                             // ready for the next launch on this stream
}

// out[0] = sum_u eq(u, x) V[u] over 2^s words (the multilinear extension of V at x); *bad |= 1 if a word is >= p
__global__ void __launch_bounds__(VT) k_v_mle(const uint64_t *__restrict__ V, uint32_t s, const uint64_t *__restrict__ x,
                                                uint64_t *part, unsigned *ticket, uint64_t *out, unsigned *bad) {
    extern __shared__ __align__(16) uint64_t vsm[];
    __shared__ uint64_t red[32], xs[MAX_VARS];
    const uint32_t tid = threadIdx.x;
    if (tid < s) xs[tid] = x[tid];
    __syncthreads();
    const EqTab e = build_eq_tab(vsm, vsm + (2u << V_EQLOG), xs, s, tid);
    __syncthreads();
    const uint64_t n = 1ull << s;
    acc128 A; A.clear();
    uint64_t sum = 0; uint32_t cnt = 0; unsigned nc = 0;
    for (uint64_t u = (uint64_t)blockIdx.x * VT + tid; u < n; u += (uint64_t)gridDim.x * VT) {
        const uint64_t w = __ldg(V + u);
        nc |= w >= fp61::P;
        A.mac(e.eq_of((uint32_t)u), w & fp61::P);
        if (++cnt == 32) { sum = fp61::add(sum, A.value()); A.clear(); cnt = 0; }
    }
    if (nc) atomicOr(bad, 1u);
    uint64_t v[1] = {fp61::add(sum, A.value())};
    verifier_reduce<1>(v, red, part, ticket, out);
}

// out[t] = sum over the gates of type t of eq(g, z) eq(in1[g], r1) eq(in2[g], r2), t = 0..3
__global__ void __launch_bounds__(VT) k_v_wiring(const uint8_t *__restrict__ type, const uint32_t *__restrict__ in1,
                                                   const uint32_t *__restrict__ in2, uint32_t si, uint32_t s,
                                                   const uint64_t *__restrict__ pts /* z[64] | r1[64] | r2[64] */,
                                                   uint64_t *part, unsigned *ticket, uint64_t *out) {
    extern __shared__ __align__(16) uint64_t vsm[];
    __shared__ uint64_t red[4 * 32], xs[3 * MAX_VARS];
    const uint32_t tid = threadIdx.x;
    if (tid < 3 * MAX_VARS) xs[tid] = pts[tid];
    __syncthreads();
    const EqTab ez = build_eq_tab(vsm, vsm + (2u << V_EQLOG), xs, si, tid);
    const EqTab e1 = build_eq_tab(vsm + V_TAB_WORDS, vsm + V_TAB_WORDS + (2u << V_EQLOG), xs + MAX_VARS, s, tid);
    const EqTab e2 = build_eq_tab(vsm + 2 * V_TAB_WORDS, vsm + 2 * V_TAB_WORDS + (2u << V_EQLOG), xs + 2 * MAX_VARS, s, tid);
    __syncthreads();
    const uint64_t n = 1ull << si;
    acc128 A[4];
    uint64_t v[4] = {0, 0, 0, 0};
#pragma unroll
    for (int t = 0; t < 4; t++) A[t].clear();
    uint32_t cnt = 0;
    for (uint64_t g = (uint64_t)blockIdx.x * VT + tid; g < n; g += (uint64_t)gridDim.x * VT) {
        const uint32_t t = __ldg(type + g);
        const uint64_t w = fp61::mul(ez.eq_of((uint32_t)g), e1.eq_of(__ldg(in1 + g)));
        const uint64_t f = e2.eq_of(__ldg(in2 + g));
        const uint64_t pl = w * f, ph = fp61::mulhi(w, f);
#pragma unroll
        for (int q = 0; q < 4; q++) if (t == (uint32_t)q) { A[q].lo += pl; A[q].hi += ph + (A[q].lo < pl); }
        if (++cnt == 32) {
#pragma unroll
            for (int q = 0; q < 4; q++) { v[q] = fp61::add(v[q], A[q].value()); A[q].clear(); }
            cnt = 0;
        }
    }
#pragma unroll
    for (int q = 0; q < 4; q++) v[q] = fp61::add(v[q], A[q].value());
    verifier_reduce<4>(v, red, part, ticket, out);
}

struct VerifierHost {                                      // per circuit, allocated on first use
    uint64_t *d_pts = nullptr, *d_res = nullptr, *d_part = nullptr;
    unsigned *d_flags = nullptr;                           // [0] ticket, [1] non-canonical word seen
    uint64_t *h_pin = nullptr;                             // transcript + results staging
    int blocks = 0;
};
static std::vector<std::pair<const vc_circuit *, VerifierHost *>> g_verifiers;   // heap entries, guarded by g_registry_mutex

static VerifierHost *verifier_of(const vc_circuit *c) {
    std::lock_guard<std::mutex> lk(g_registry_mutex);
    for (auto &p : g_verifiers) if (p.first == c) return p.second;
    VerifierHost v;
    v.blocks = std::min(V_MAX_BLOCKS, 2 * c->sm_count);
    const size_t npts = (size_t)(c->d + 2) * 3 * MAX_VARS, nres = 4 * (size_t)c->d + 2;
    if (cudaMalloc(&v.d_pts, npts * 8) != cudaSuccess || cudaMalloc(&v.d_res, nres * 8) != cudaSuccess ||
        cudaMalloc(&v.d_part, (size_t)V_MAX_BLOCKS * 4 * 8) != cudaSuccess || cudaMalloc(&v.d_flags, 2 * sizeof(unsigned)) != cudaSuccess ||
        cudaMallocHost(&v.h_pin, (c->total_words + nres + npts + 2) * 8) != cudaSuccess) {
        (void)cudaGetLastError();
        cudaFree(v.d_pts); cudaFree(v.d_res); cudaFree(v.d_part); cudaFree(v.d_flags);
        if (v.h_pin) cudaFreeHost(v.h_pin);
        return nullptr;
    }
    cudaFuncSetAttribute(k_v_mle, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(V_TAB_WORDS * 8));
    cudaFuncSetAttribute(k_v_wiring, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(3 * V_TAB_WORDS * 8));
    VerifierHost *hv = new (std::nothrow) VerifierHost(v);
    if (!hv) { cudaFree(v.d_pts); cudaFree(v.d_res); cudaFree(v.d_part); cudaFree(v.d_flags); cudaFreeHost(v.h_pin); return nullptr; }
    g_verifiers.emplace_back(c, hv);
    return hv;
}

void verifier_free(const vc_circuit *c) {
    std::lock_guard<std::mutex> lk(g_registry_mutex);
    for (size_t i = 0; i < g_verifiers.size(); i++)
        if (g_verifiers[i].first == c) {
            VerifierHost &v = *g_verifiers[i].second;
            cudaFree(v.d_pts); cudaFree(v.d_res); cudaFree(v.d_part); cudaFree(v.d_flags); cudaFreeHost(v.h_pin);
            delete g_verifiers[i].second;
            g_verifiers.erase(g_verifiers.begin() + i);
            return;
        }
}

}  // namespace vc

namespace {
using u64 = uint64_t;
// the host side of the checks: closed forms written for this file (vc_verify.cu has its own)
u64 quad_at(const u64 *G, u64 r) {                         // the quadratic through (0,G0),(1,G1),(2,G2) at r
    const u64 half = 1ull << 60, a = fp61::sub(r, 1), b = fp61::sub(r, 2);
    u64 acc = fp61::mul(G[0], fp61::mul(fp61::mul(a, b), half));
    acc = fp61::sub(acc, fp61::mul(G[1], fp61::mul(r, b)));
    return fp61::add(acc, fp61::mul(G[2], fp61::mul(fp61::mul(r, a), half)));
}
u64 power(u64 a, u64 e) { u64 r = 1; for (; e; e >>= 1, a = fp61::mul(a, a)) if (e & 1) r = fp61::mul(r, a); return r; }
// degree <= s through (k, q[k]), k = 0..s, at tau: sum_k q[k] prod_{m != k}(tau - m) / (k! (s-k)! (-1)^(s-k)); the products
// come from prefix and suffix tables, invf[k] = 1/k! from one inversion per call of the verifier
u64 poly_at(const u64 *q, uint32_t s, u64 tau, const std::vector<u64> &invf) {
    std::vector<u64> pre(s + 2), suf(s + 2);
    pre[0] = 1; suf[s + 1] = 1;
    for (uint32_t k = 0; k <= s; k++) pre[k + 1] = fp61::mul(pre[k], fp61::sub(tau, k));
    for (uint32_t k = s + 1; k-- > 0;) suf[k] = fp61::mul(suf[k + 1], fp61::sub(tau, k));
    u64 tot = 0;
    for (uint32_t k = 0; k <= s; k++) {
        const u64 t = fp61::mul(fp61::mul(q[k], fp61::mul(pre[k], suf[k + 1])), fp61::mul(invf[k], invf[s - k]));
        tot = ((s - k) & 1) ? fp61::sub(tot, t) : fp61::add(tot, t);
    }
    return tot;
}
u64 apply_gate(uint32_t t, u64 L, u64 R) { return t == VC_ADD ? fp61::add(L, R) : t == VC_MULT ? fp61::mul(L, R) : t == VC_SUB ? fp61::sub(L, R) : L; }
}  // namespace

extern "C" int vc_verify_transcript_device(const vc_circuit *c, const uint64_t *d_input, const uint64_t *d_outputs, uint64_t seed,
                                           const uint64_t *d_transcript, uint64_t n_words, int *accept, uint32_t *fail_layer,
                                           uint32_t *fail_round, void *cuda_stream) {
    using namespace vc;
    if (!c || !d_input || !d_outputs || !d_transcript || !accept || !fail_layer || !fail_round) return VC_ERR_ARG;
    *accept = 0; *fail_layer = 0; *fail_round = 0;
    if (n_words != c->total_words) return VC_ERR_ARG;
    if (c->hosted) return VC_ERR_STATE;                        // the wiring sums read device-resident records; a hosted circuit has none
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { (void)cudaGetLastError(); return VC_ERR_CUDA; }
    VerifierHost *vh = verifier_of(c);
    if (!vh) return VC_ERR_NOMEM;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const uint32_t d = c->d;
    const size_t npts = (size_t)(d + 2) * 3 * MAX_VARS, nres = 4 * (size_t)d + 2;
    u64 *h_tr = vh->h_pin, *h_res = h_tr + c->total_words, *h_pts = h_res + nres;
    unsigned *h_flags = reinterpret_cast<unsigned *>(h_pts + npts);
    // ---- every point of the protocol from the seed alone: z_0, then per layer (r1, r2, tau) and z_{i+1} = l(tau)
    std::memset(h_pts, 0, npts * 8);
    std::vector<u64> taus(d);
    u64 ctr = 0;
    u64 *z = h_pts;                                            // block i: z_i | r1_i | r2_i
    for (uint32_t k = 0; k < c->logs[0]; k++) z[k] = fp61::draw(seed, ctr++);
    for (uint32_t i = 0; i < d; i++) {
        const uint32_t s = c->logs[i + 1];
        u64 *blk = h_pts + (size_t)i * 3 * MAX_VARS, *r1 = blk + MAX_VARS, *r2 = blk + 2 * MAX_VARS, *zn = blk + 3 * MAX_VARS;
        if (i == 0 && c->sum_out) {              // the sum gate: s draws, and they ARE the next point (no r2, no tau)
            for (uint32_t k = 0; k < s; k++) zn[k] = r1[k] = fp61::draw(seed, ctr++);
            continue;
        }
        for (uint32_t k = 0; k < s; k++) r1[k] = fp61::draw(seed, ctr++);
        for (uint32_t k = 0; k < s; k++) r2[k] = fp61::draw(seed, ctr++);
        taus[i] = fp61::draw(seed, ctr++);
        for (uint32_t k = 0; k < s; k++) zn[k] = fp61::add(r1[k], fp61::mul(taus[i], fp61::sub(r2[k], r1[k])));
    }
    // ---- enqueue: points up, the d + 2 sums, results and transcript down
    if (cudaMemcpyAsync(vh->d_pts, h_pts, npts * 8, cudaMemcpyHostToDevice, st) != cudaSuccess) return VC_ERR_CUDA;
    if (cudaMemsetAsync(vh->d_flags, 0, 2 * sizeof(unsigned), st) != cudaSuccess) return VC_ERR_CUDA;
    auto blocks_for = [&](uint64_t n) { return (unsigned)std::max<uint64_t>(1, std::min<uint64_t>((n + VT - 1) / VT, (uint64_t)vh->blocks)); };
    VC_LAUNCH(VC_K_MISC, k_v_mle, blocks_for(1ull << c->logs[0]), VT, V_TAB_WORDS * 8, st, d_outputs, c->logs[0], vh->d_pts, vh->d_part,
              vh->d_flags, vh->d_res, vh->d_flags + 1);
    if (c->sum_out && cudaMemsetAsync(vh->d_res + 1, 0, 4 * 8, st) != cudaSuccess) return VC_ERR_CUDA;   // no wiring sums for the sum gate
    for (uint32_t i = c->first_pair_layer(); i < d; i++)
        VC_LAUNCH(VC_K_MISC, k_v_wiring, blocks_for(1ull << c->logs[i]), VT, 3 * V_TAB_WORDS * 8, st, c->d_type[i], c->d_in1[i], c->d_in2[i],
                  c->logs[i], c->logs[i + 1], vh->d_pts + (size_t)i * 3 * MAX_VARS, vh->d_part, vh->d_flags, vh->d_res + 1 + 4 * (size_t)i);
    VC_LAUNCH(VC_K_MISC, k_v_mle, blocks_for(1ull << c->log_input), VT, V_TAB_WORDS * 8, st, d_input, c->log_input,
              vh->d_pts + (size_t)d * 3 * MAX_VARS, vh->d_part, vh->d_flags, vh->d_res + 1 + 4 * (size_t)d, vh->d_flags + 1);
    if (cudaGetLastError() != cudaSuccess) return VC_ERR_CUDA;
    if (cudaMemcpyAsync(h_res, vh->d_res, nres * 8, cudaMemcpyDeviceToHost, st) != cudaSuccess) return VC_ERR_CUDA;
    if (cudaMemcpyAsync(h_flags, vh->d_flags, 2 * sizeof(unsigned), cudaMemcpyDeviceToHost, st) != cudaSuccess) return VC_ERR_CUDA;
    if (cudaMemcpyAsync(h_tr, d_transcript, n_words * 8, cudaMemcpyDeviceToHost, st) != cudaSuccess) return VC_ERR_CUDA;
    if (cudaStreamSynchronize(st) != cudaSuccess) { (void)cudaGetLastError(); return VC_ERR_CUDA; }
    if (h_flags[1]) return VC_ERR_ARG;                         // non-canonical input or output word
    for (u64 w = 0; w < n_words; w++) if (h_tr[w] >= fp61::P) return VC_ERR_ARG;
    // ---- the O(rounds) checks, in protocol order
    uint32_t smax = 1;
    for (uint32_t i = 1; i <= d; i++) smax = std::max(smax, c->logs[i]);
    std::vector<u64> invf(smax + 1);
    {
        u64 fact = 1;
        for (uint32_t k = 2; k <= smax; k++) fact = fp61::mul(fact, k);
        u64 inv = power(fact, fp61::P - 2);
        for (uint32_t k = smax; k >= 1; k--) { invf[k] = inv; inv = fp61::mul(inv, k); }
        invf[0] = 1;
    }
    u64 claim = h_res[0];
    const u64 *tr = h_tr;
    for (uint32_t i = 0; i < d; i++) {
        const uint32_t s = c->logs[i + 1];
        const u64 *blk = h_pts + (size_t)i * 3 * MAX_VARS;
        if (i == 0 && c->sum_out) {
            for (uint32_t m = 0; m < s; m++, tr += 2) {
                if (fp61::add(tr[0], tr[1]) != claim) { *fail_layer = 0; *fail_round = m; return VC_OK; }
                claim = fp61::add(tr[0], fp61::mul(blk[MAX_VARS + m], fp61::sub(tr[1], tr[0])));
            }
            continue;
        }
        for (uint32_t m = 0; m < 2 * s; m++, tr += 3) {
            if (fp61::add(tr[0], tr[1]) != claim) { *fail_layer = i; *fail_round = m; return VC_OK; }
            claim = quad_at(tr, m < s ? blk[MAX_VARS + m] : blk[2 * MAX_VARS + (m - s)]);
        }
        const u64 *q = tr; tr += s + 1;
        const u64 *W = h_res + 1 + 4 * (size_t)i;
        u64 rhs = 0;
        for (uint32_t t = 0; t < 4; t++) rhs = fp61::add(rhs, fp61::mul(W[t], apply_gate(t, q[0], q[1])));
        if (rhs != claim) { *fail_layer = i; *fail_round = 2 * s; return VC_OK; }
        claim = poly_at(q, s, taus[i], invf);
    }
    if (h_res[1 + 4 * (size_t)d] != claim) { *fail_layer = d; *fail_round = 0; return VC_OK; }
    *accept = 1;
    return VC_OK;
}

/* debug: the device sums of the last vc_verify_transcript_device call: [0] start claim, [1 + 4 i + t] wiring sum of
 * type t of layer i, [1 + 4 d] the closing input extension */
extern "C" int vc_debug_verifier_sums(const vc_circuit *c, uint64_t *h_sums, uint64_t n) {
    if (!c || !h_sums || n != 4 * (uint64_t)c->d + 2) return VC_ERR_ARG;
    std::lock_guard<std::mutex> lk(vc::g_registry_mutex);
    for (auto &p : vc::g_verifiers)
        if (p.first == c) { std::memcpy(h_sums, p.second->h_pin + c->total_words, n * 8); return VC_OK; }
    return VC_ERR_STATE;
}

namespace vc {
// ------------------------------------------------------------------------------------------------------------------
// vc_mle_device_noalloc — the multilinear extension of a device table at one point (the verifier's "secret", PAPER.md:127
// §4.1.2: one chi-weighted term per element, reduced in F_p) for callers that cannot allocate: code under CUDA graph
// capture, tight serving loops, harnesses that forbid cudaMalloc.  Same arithmetic as k_v_mle above; what differs is
// where the kernel's scratch lives: the block partials, the last-block ticket and the status word sit in ONE file-scope
// device array of fixed size instead of the per-circuit cudaMalloc'd scratch of verifier_of().  Every GPU that loads the
// library holds these VC_NOALLOC_SCRATCH_WORDS * 8 = 4 KB until the process exits.
//
// In host code `g_noalloc_scratch` is a host-side stand-in, not a device address, so the host never passes the name to a
// kernel: once per device, with that device current, noalloc_scratch() asks cudaGetSymbolAddress for the address and keeps it.
// Every call on a device shares the array and finds the previous call's contents in it: the ticket and status words are
// cleared on the caller's stream before each launch (the partials are rewritten before they are read).  Calls that
// overlap on the GPU (two streams, two host threads) race on the array: serialise them.
constexpr uint32_t NA_PART = 0;                           // [0, V_MAX_BLOCKS): one partial per block
constexpr uint32_t NA_TICKET = V_MAX_BLOCKS;              // low 32 bits: last-block ticket
constexpr uint32_t NA_BAD = V_MAX_BLOCKS + 1;             // low 32 bits: 1 = a word >= p was seen
static_assert(NA_BAD < VC_NOALLOC_SCRATCH_WORDS, "scratch array too small for the partials");
static __device__ __align__(256) unsigned long long g_noalloc_scratch[VC_NOALLOC_SCRATCH_WORDS];

// k_v_mle with its scratch taken from one array: out[0] = sum_u eq(u, x) V[u] over 2^s words
__global__ void __launch_bounds__(VT) k_v_mle_static(const uint64_t *__restrict__ V, uint32_t s, const uint64_t *__restrict__ x,
                                                       unsigned long long *scratch, uint64_t *out) {
    extern __shared__ __align__(16) uint64_t vsm[];
    __shared__ uint64_t red[32], xs[MAX_VARS];
    uint64_t *part = reinterpret_cast<uint64_t *>(scratch + NA_PART);
    unsigned *ticket = reinterpret_cast<unsigned *>(scratch + NA_TICKET), *bad = reinterpret_cast<unsigned *>(scratch + NA_BAD);
    const uint32_t tid = threadIdx.x;
    if (tid < s) xs[tid] = x[tid];
    __syncthreads();
    const EqTab e = build_eq_tab(vsm, vsm + (2u << V_EQLOG), xs, s, tid);
    __syncthreads();
    const uint64_t n = 1ull << s;
    acc128 A; A.clear();
    uint64_t sum = 0; uint32_t cnt = 0; unsigned nc = 0;
    for (uint64_t u = (uint64_t)blockIdx.x * VT + tid; u < n; u += (uint64_t)gridDim.x * VT) {
        const uint64_t w = __ldg(V + u);
        nc |= w >= fp61::P;
        A.mac(e.eq_of((uint32_t)u), w & fp61::P);
        if (++cnt == 32) { sum = fp61::add(sum, A.value()); A.clear(); cnt = 0; }
    }
    if (nc) atomicOr(bad, 1u);
    uint64_t v[1] = {fp61::add(sum, A.value())};
    verifier_reduce<1>(v, red, part, ticket, out);
}

constexpr int NA_MAX_DEVICES = 64;
static unsigned long long *g_noalloc_ptr[NA_MAX_DEVICES];  // per device: the array's DEVICE address (null: not asked yet)
static std::mutex g_noalloc_mutex;

// set-up, once per device, with that device current: the device address of the scratch array
static int noalloc_scratch(unsigned long long **p) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= NA_MAX_DEVICES) { (void)cudaGetLastError(); return VC_ERR_CUDA; }
    std::lock_guard<std::mutex> lk(g_noalloc_mutex);
    if (!g_noalloc_ptr[dev]) {
        unsigned long long *q = nullptr;
        if (cudaGetSymbolAddress((void **)&q, g_noalloc_scratch) != cudaSuccess || !q) { (void)cudaGetLastError(); return VC_ERR_CUDA; }
        g_noalloc_ptr[dev] = q;
    }
    *p = g_noalloc_ptr[dev];
    return VC_OK;
}

}  // namespace vc

extern "C" int vc_mle_device_noalloc(const uint64_t *d_values, uint32_t log_n, const uint64_t *d_point, uint64_t *d_out2,
                                     void *cuda_stream) {
    using namespace vc;
    if (!d_values || !d_out2 || (log_n > 0 && !d_point)) return VC_ERR_ARG;
    if (log_n > VC_NOALLOC_MAX_LOG) return VC_ERR_LIMIT;       // beyond the stated maximum: nothing is enqueued
    unsigned long long *scr = nullptr;
    const int rc = noalloc_scratch(&scr);
    if (rc != VC_OK) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // the array keeps the last call's contents: ticket and status start at zero (adjacent words: one memset node)
    if (cudaMemsetAsync(scr + NA_TICKET, 0, 2 * sizeof(unsigned long long), st) != cudaSuccess) { (void)cudaGetLastError(); return VC_ERR_CUDA; }
    const uint64_t n = 1ull << log_n;
    const unsigned blocks = (unsigned)std::max<uint64_t>(1, std::min<uint64_t>((n + VT - 1) / VT, (uint64_t)V_MAX_BLOCKS));
    k_v_mle_static<<<blocks, VT, V_TAB_WORDS * 8, st>>>(d_values, log_n, d_point, scr, d_out2);   // (not VC_LAUNCH: its profiling mode creates events)
    g_launches.fetch_add(1, std::memory_order_relaxed);
    if (cudaGetLastError() != cudaSuccess) return VC_ERR_CUDA;
    // d_out2[1] <- the status word (0 / 1), device to device on the same stream
    if (cudaMemcpyAsync(d_out2 + 1, scr + NA_BAD, sizeof(unsigned long long), cudaMemcpyDeviceToDevice, st) != cudaSuccess) { (void)cudaGetLastError(); return VC_ERR_CUDA; }
    return VC_OK;
}
