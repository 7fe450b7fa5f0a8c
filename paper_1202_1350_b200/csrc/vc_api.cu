// vc_api.cu — host side of libvc.so: load / evaluate / prove_layer (streaming schedule) / helpers.
// C ABI documented in include/vc.h.  PyTorch is not involved here: plain CUDA runtime, caller's stream.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdlib>
#include <cstring>
#include <new>

#include "vc_circuit.hpp"
#include "vc_kernels.cuh"
#include "vc_line.cuh"
#include "vc_round.cuh"
#include "vc_sum.cuh"

namespace vc {
std::atomic<uint64_t> g_launches{0};
bool g_profile = false;
std::vector<ProfRec> g_prof;
std::mutex g_registry_mutex;
void prof_push(int kind, cudaEvent_t a, cudaEvent_t b) { std::lock_guard<std::mutex> lk(g_registry_mutex); g_prof.push_back({kind, a, b}); }
}

#define CUDA_TRY(x)                                          \
    do {                                                     \
        cudaError_t e_ = (x);                                \
        if (e_ != cudaSuccess) {                             \
            (void)cudaGetLastError();                        \
            return e_ == cudaErrorMemoryAllocation ? VC_ERR_NOMEM : VC_ERR_CUDA; \
        }                                                    \
    } while (0)

static inline uint32_t grid_for(uint64_t n, int sm_count, int per_thread = 4) {
    uint64_t b = (n + (uint64_t)vc::RED_BLOCK * per_thread - 1) / ((uint64_t)vc::RED_BLOCK * per_thread);
    uint64_t cap = (uint64_t)sm_count * 4;
    if (b < 1) b = 1;
    if (b > cap) b = cap;
    return (uint32_t)b;
}

static uint64_t host_pow(uint64_t a, uint64_t e) {
    uint64_t r = 1;
    while (e) { if (e & 1) r = fp61::mul(r, a); a = fp61::mul(a, a); e >>= 1; }
    return r;
}

extern "C" const char *vc_strerror(int code) {
    switch (code) {
    case VC_OK: return "ok";
    case VC_ERR_ARG: return "bad argument";
    case VC_ERR_SHAPE: return "bad circuit shape (non power of two, index out of range, unknown gate type, or a layer below of size 1)";
    case VC_ERR_STATE: return "call out of order (vc_evaluate, then vc_prove_layer 0..d-1 with one seed)";
    case VC_ERR_CUDA: return "CUDA error (no device, launch or copy failure)";
    case VC_ERR_NOMEM: return "out of memory";
    case VC_ERR_LIMIT: return "size beyond the fixed maximum of an entry point that allocates nothing (vc_mle_device_noalloc: log_n <= 28)";
    default: return "unknown error";
    }
}

extern "C" void vc_circuit_free(vc_circuit *c) {
    if (!c) return;
    vc::fused_free(c);
    vc::verifier_free(c);
    vc::hosted_free(c);
    for (auto p : c->d_type) cudaFree(p);
    for (auto p : c->d_in1) cudaFree(p);
    for (auto p : c->d_in2) cudaFree(p);
    for (auto p : c->d_V) cudaFree(p);
    cudaFree(c->d_P); cudaFree(c->d_T0); cudaFree(c->d_T1); cudaFree(c->d_part); cudaFree(c->d_tr);
    cudaFree(c->d_state);
    delete c;
}

// Fits the bit-field rule of vc_state.cuh to one index array: c = f(0), w_p = f(2^p) - c; every non-zero w_p must be a power
// of two and consecutive bits with doubling weights form a field (at most three); the rule is then verified on every gate.
static bool fit_index_rule(const uint32_t *f, uint32_t log_n, uint32_t &mask, uint32_t &c, vc::WireField (&fl)[3]) {
    c = f[0];
    uint32_t top = 0;
    for (uint64_t g = 0; g < (1ull << log_n); g++) top |= f[g];
    mask = 1; while (mask < top) mask = 2 * mask + 1;          // indices wrap at the smallest power of two above them
    uint32_t nf = 0;
    uint32_t p = 0;
    while (p < log_n) {
        const uint32_t w = (f[1u << p] - c) & mask;
        if (w == 0) { p++; continue; }
        if (w & (w - 1)) return false;
        uint32_t q0 = 0; while ((1u << q0) != w) q0++;
        uint32_t len = 1;
        while (p + len < log_n && q0 + len < 32 && ((f[1u << (p + len)] - c) & mask) == (w << len)) len++;
        if (nf == 3) return false;
        fl[nf].p0 = p; fl[nf].m = (uint32_t)((1ull << len) - 1); fl[nf].q0 = q0; fl[nf].pad = 0; nf++;
        p += len;
    }
    const uint64_t n = 1ull << log_n;
    for (uint64_t g = 0; g < n; g++) {
        uint32_t v = c;
        for (uint32_t k = 0; k < 3; k++) v += (((uint32_t)g >> fl[k].p0) & fl[k].m) << fl[k].q0;
        if ((v & mask) != f[g]) return false;
    }
    return true;
}
static bool fit_wire_rule(const vc_layer &L, uint32_t log_below, vc::WireRule &r) {
    const uint32_t ln = L.log_size;
    if (ln == 0 || log_below > 31) return false;
    const uint64_t n = 1ull << ln;
    r = vc::WireRule{};
    r.t[0] = L.type[0]; r.t[1] = L.type[n - 1]; r.tbit = 0; r.tm = 0;
    bool one = true, lanes = true;
    for (uint64_t g = 0; g < n; g++) {
        one = one && L.type[g] == r.t[0];
        lanes = lanes && L.type[g] == r.t[(g >> (ln - 1)) & 1];
    }
    if (!one) { if (!lanes) return false; r.tbit = ln - 1; r.tm = 1; }
    return fit_index_rule(L.in1, ln, r.mask[0], r.c[0], r.f[0]) && fit_index_rule(L.in2, ln, r.mask[1], r.c[1], r.f[1]);
}

static int load_impl(const vc_layer *layers, uint32_t d, uint32_t log_input, vc_circuit *c) {
    int dev = 0, ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { (void)cudaGetLastError(); return VC_ERR_CUDA; }
    CUDA_TRY(cudaGetDevice(&dev));
    CUDA_TRY(cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, dev));
    CUDA_TRY(cudaDeviceGetAttribute(&c->coop_ok, cudaDevAttrCooperativeLaunch, dev));
    c->d = d; c->log_input = log_input;
    c->logs.resize(d + 1);
    for (uint32_t i = 0; i < d; i++) c->logs[i] = layers[i].log_size;
    c->logs[d] = log_input;
    for (uint32_t i = 0; i <= d; i++) if (c->logs[i] > 30) return VC_ERR_SHAPE;
    for (uint32_t i = 1; i <= d; i++) if (c->logs[i] == 0) return VC_ERR_SHAPE;   // a layer below of size 1
    c->h_type.resize(d); c->h_in1.resize(d); c->h_in2.resize(d); c->wiring.assign(d, 0); c->wrule.assign(d, vc::WireRule{});
    uint64_t max_gates = 1, max_tab = 2, total = 0;
    size_t part = (size_t)vc::MAX_PART_BLOCKS * 3;
    for (uint32_t i = 0; i < d; i++) {
        const vc_layer &L = layers[i];
        if (!L.type || !L.in1 || !L.in2) return VC_ERR_ARG;
        const uint64_t n = 1ull << L.log_size, nb = 1ull << c->logs[i + 1];
        bool tree = true, self = true, onetype = true;
        if (i == 0 && L.log_size == 0 && L.type[0] == VC_SUM) c->sum_out = true;    // the one sum gate over all of layer 1: in1 / in2 are not read
        for (uint64_t g = 0; g < n && !(i == 0 && c->sum_out); g++) {
            if (L.type[g] > 3 || L.in1[g] >= nb || L.in2[g] >= nb) return VC_ERR_SHAPE;
            tree = tree && L.in1[g] == 2 * g && L.in2[g] == 2 * g + 1;
            self = self && L.in1[g] == g && L.in2[g] == g;
            onetype = onetype && L.type[g] == L.type[0];
        }
        c->wiring[i] = !onetype ? 0u : (tree ? 1u : (self ? 2u : 0u));
        if (i == 0 && c->sum_out) c->wiring[i] = 0u;
        const bool no_rule = getenv("VC_NO_WIRE_RULE") != nullptr;     // read at every load: records are read unless tree / self
        if (c->wiring[i] == 0 && !no_rule && !(i == 0 && c->sum_out) && fit_wire_rule(L, c->logs[i + 1], c->wrule[i])) c->wiring[i] = 3u;
        c->h_type[i].assign(L.type, L.type + n);
        c->h_in1[i].assign(L.in1, L.in1 + n);
        c->h_in2[i].assign(L.in2, L.in2 + n);
        max_gates = std::max(max_gates, n);
        max_tab = std::max(max_tab, nb);
        const uint32_t s = c->logs[i + 1];
        total += c->layer_words(i);
        const uint32_t used = std::min<uint32_t>(s, vc::LINE_NT + vc::LINE_TB);
        part = std::max(part, (size_t)(1ull << (s - used)) * (s > 1 ? s - 1 : 1));
    }
    c->total_words = total;
    c->part_words = part;
    c->d_type.assign(d, nullptr); c->d_in1.assign(d, nullptr); c->d_in2.assign(d, nullptr);
    c->d_V.assign(d + 1, nullptr);
    for (uint32_t i = 0; i < d && !c->hosted; i++) {     // hosted: the records never live on the device as a whole (vc_hosted.cu)
        const size_t n = (size_t)1 << c->logs[i];
        CUDA_TRY(cudaMalloc(&c->d_type[i], n));
        CUDA_TRY(cudaMalloc(&c->d_in1[i], n * 4));
        CUDA_TRY(cudaMalloc(&c->d_in2[i], n * 4));
        CUDA_TRY(cudaMemcpy(c->d_type[i], layers[i].type, n, cudaMemcpyHostToDevice));
        CUDA_TRY(cudaMemcpy(c->d_in1[i], layers[i].in1, n * 4, cudaMemcpyHostToDevice));
        CUDA_TRY(cudaMemcpy(c->d_in2[i], layers[i].in2, n * 4, cudaMemcpyHostToDevice));
    }
    for (uint32_t i = 0; i <= d; i++) CUDA_TRY(cudaMalloc(&c->d_V[i], (size_t)8 << c->logs[i]));
    if (!c->hosted) CUDA_TRY(cudaMalloc(&c->d_P, max_gates * 8));     // hosted: the weights live in pinned host memory
    CUDA_TRY(cudaMalloc(&c->d_T0, std::max<uint64_t>(max_tab / 2, 2) * 8));
    CUDA_TRY(cudaMalloc(&c->d_T1, std::max<uint64_t>(max_tab / 4, 2) * 8));
    CUDA_TRY(cudaMalloc(&c->d_part, part * 8));
    CUDA_TRY(cudaMalloc(&c->d_tr, total * 8));
    CUDA_TRY(cudaMalloc(&c->d_state, sizeof(vc::DevState)));
    // proof state: zero, plus 1/k! for the Lagrange denominators (constants of the method, not data)
    vc::DevState *hs = new (std::nothrow) vc::DevState();
    if (!hs) return VC_ERR_NOMEM;
    std::memset(hs, 0, sizeof(*hs));
    uint64_t fact = 1;
    for (uint32_t k = 1; k <= vc::MAX_VARS; k++) fact = fp61::mul(fact, k);
    uint64_t inv = host_pow(fact, fp61::P - 2);
    for (int k = vc::MAX_VARS; k >= 0; k--) { hs->invfact[k] = inv; inv = fp61::mul(inv, (uint64_t)k); }
    cudaError_t e = cudaMemcpy(c->d_state, hs, sizeof(*hs), cudaMemcpyHostToDevice);
    delete hs;
    CUDA_TRY(e);
    CUDA_TRY(cudaFuncSetAttribute(vc::k_line, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024));
    if (c->hosted) { c->schedule = 2; return vc::hosted_init(c); }
    return vc::fused_init(c);
}

static int load_any(const vc_layer *layers, uint32_t d, uint32_t log_input, bool hosted, uint32_t chunk_log, vc_circuit **out);
extern "C" int vc_circuit_load(const vc_layer *layers, uint32_t d, uint32_t log_input, vc_circuit **out) {
    return load_any(layers, d, log_input, false, 0, out);
}
extern "C" int vc_circuit_load_hosted(const vc_layer *layers, uint32_t d, uint32_t log_input, uint32_t chunk_log, vc_circuit **out) {
    if (chunk_log < 8 || chunk_log > 28) return VC_ERR_ARG;
    return load_any(layers, d, log_input, true, chunk_log, out);
}
extern "C" int vc_hosted_set_weights(vc_circuit *c, int swap) {
    if (!c || swap < 0 || swap > 1) return VC_ERR_ARG;
    if (!c->hosted) return VC_ERR_STATE;
    c->hosted_swap = swap != 0;
    return VC_OK;
}
extern "C" int vc_debug_hosted_bytes(const vc_circuit *c, uint64_t *h2d, uint64_t *d2h) {
    if (!c || !h2d || !d2h) return VC_ERR_ARG;
    if (!c->hosted) return VC_ERR_STATE;
    *h2d = c->h2d_bytes; *d2h = c->d2h_bytes;
    return VC_OK;
}
static int load_any(const vc_layer *layers, uint32_t d, uint32_t log_input, bool hosted, uint32_t chunk_log, vc_circuit **out) {
    if (!layers || !out || d == 0) return VC_ERR_ARG;
    *out = nullptr;
    vc_circuit *c = new (std::nothrow) vc_circuit();
    if (!c) return VC_ERR_NOMEM;
    c->hosted = hosted; c->chunk_log = chunk_log;
    int rc;
    try { rc = load_impl(layers, d, log_input, c); } catch (const std::bad_alloc &) { rc = VC_ERR_NOMEM; }
    if (rc != VC_OK) { vc_circuit_free(c); return rc; }
    *out = c;
    return VC_OK;
}

// ------------------------------------------------------------------ a1
extern "C" int vc_evaluate(vc_circuit *c, const uint64_t *d_input, uint64_t *d_outputs, void *cuda_stream) {
    if (!c || !d_input) return VC_ERR_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const uint32_t d = c->d;
    const uint64_t n_in = 1ull << c->log_input;
    CUDA_TRY(cudaMemsetAsync(&c->d_state->flags, 0, 2 * sizeof(unsigned int), st));   // the status word reports THIS evaluation; + k_eval_all's counter
    if (c->hosted) {
        const int rc = vc::hosted_evaluate(c, d_input, d_outputs, st);
        if (rc == VC_OK) c->next_layer = 0;
        return rc;
    }
    if (c->schedule != 1) {                      // one cooperative launch for the whole evaluation when the circuit allows it
        int rc = vc::enqueue_eval_fused(c, d_input, d_outputs, st);
        if (rc == VC_OK && c->sum_out) rc = vc::enqueue_sum_eval(c, d_outputs, st);
        if (rc == VC_OK) { c->next_layer = 0; return VC_OK; }
        if (rc != VC_ERR_STATE) return rc;
    }
    VC_LAUNCH(VC_K_EVAL, vc::k_copy_input, grid_for(n_in, c->sm_count), vc::RED_BLOCK, 0, st, d_input, c->d_V[d], n_in, c->d_state);
    for (int i = (int)d - 1; i >= (int)c->first_pair_layer(); i--) {
        const uint32_t n = 1u << c->logs[i];
        VC_LAUNCH(VC_K_EVAL, vc::k_eval, grid_for(n, c->sm_count, 2), vc::RED_BLOCK, 0, st, c->d_type[i], c->d_in1[i], c->d_in2[i],
                  c->d_V[i + 1], c->d_V[i], (i == 0 ? d_outputs : (uint64_t *)nullptr), n);
    }
    CUDA_TRY(cudaGetLastError());
    if (c->sum_out) { const int rc = vc::enqueue_sum_eval(c, d_outputs, st); if (rc != VC_OK) return rc; }
    c->next_layer = 0;
    return VC_OK;
}

// ------------------------------------------------------------------ the sum gate of large fan-in at the output (vc_sum.cuh)
int vc::enqueue_sum_eval(vc_circuit *c, uint64_t *d_outputs, cudaStream_t st) {
    const uint64_t n = 1ull << c->logs[1];
    if (cudaMemsetAsync(&c->d_state->ticket, 0, sizeof(unsigned int), st) != cudaSuccess) { (void)cudaGetLastError(); return VC_ERR_CUDA; }
    VC_LAUNCH(VC_K_EVAL, vc::k_sum_eval, grid_for(n, c->sm_count), vc::RED_BLOCK, 0, st, c->d_V[1], n, c->d_V[0], d_outputs, c->d_part, c->d_state);
    return cudaGetLastError() == cudaSuccess ? VC_OK : VC_ERR_CUDA;
}

// layer 0 of a sum-gate circuit: s rounds, one pass over the folded table per round (the fold of round j and the sums of
// round j+1 share it), the last rounds in one CTA; leaves z = r, claim = V~_1(r), ctr = s for layer 1
int vc::enqueue_sum_layer(vc_circuit *c, uint64_t seed, uint64_t *d_tr, cudaStream_t st) {
    const uint32_t s = c->logs[1];
    const uint64_t n = 1ull << s;
    vc::DevState *S = c->d_state;
    if (cudaMemsetAsync(&S->ticket, 0, sizeof(unsigned int), st) != cudaSuccess) { (void)cudaGetLastError(); return VC_ERR_CUDA; }
    VC_LAUNCH(VC_K_ROUND, vc::k_sum_first, grid_for(n / 2, c->sm_count), vc::RED_BLOCK, 0, st, c->d_V[1], n, seed, c->d_part, S, d_tr);
    const uint64_t *tab = c->d_V[1];
    uint32_t j = 0;
    for (; s - j > vc::SUM_TAIL_LOG; j++) {              // tab holds 2^(s-j) words, message j is out, r_j is drawn
        uint64_t *out = (j & 1) ? c->d_T1 : c->d_T0;
        const uint64_t half = n >> (j + 1);
        VC_LAUNCH(VC_K_ROUND, vc::k_sum_fold, grid_for(half / 2, c->sm_count), vc::RED_BLOCK, 0, st, tab, out, half, j, c->d_part, S, d_tr);
        tab = out;
    }
    VC_LAUNCH(VC_K_ROUND, vc::k_sum_tail, 1, vc::SUM_TAIL_T, 0, st, tab, s - j, j, S, d_tr);
    return cudaGetLastError() == cudaSuccess ? VC_OK : VC_ERR_CUDA;
}

// ------------------------------------------------------------------ a2-a7, streaming schedule
int vc::enqueue_layer_streaming(vc_circuit *c, uint32_t layer, uint64_t seed, uint64_t *d_tr, cudaStream_t st) {
    const uint32_t si = c->logs[layer], s = c->logs[layer + 1];
    const uint32_t n = 1u << si;
    vc::DevState *S = c->d_state;
    const uint8_t *type = c->d_type[layer];
    const uint32_t *in1 = c->d_in1[layer], *in2 = c->d_in2[layer];
    const uint64_t *Vb = c->d_V[layer + 1];
    const uint32_t gg = grid_for(n, c->sm_count);
    const uint32_t cb = si < (uint32_t)vc::BETA_LOG_CHUNK ? si : (uint32_t)vc::BETA_LOG_CHUNK;
    if (layer == 0) VC_LAUNCH(VC_K_SETUP, vc::k_start, 1, 64, 0, st, S, seed, si);
    VC_LAUNCH(VC_K_SETUP, vc::k_beta, 1u << (si - cb), 256, 0, st, S, c->d_P, si);
    if (layer == 0) VC_LAUNCH(VC_K_SETUP, vc::k_dot_claim, gg, vc::RED_BLOCK, 0, st, c->d_P, c->d_V[0], n, c->d_part, S);
    uint64_t *tr = d_tr;
    for (int phase = 1; phase <= 2; phase++) {
        const uint64_t *tab = Vb;
        for (uint32_t j = 0; j < s; j++) {
            uint64_t *out = (j & 1) ? c->d_T1 : c->d_T0;
            const uint32_t half = 1u << (s - j - 1);
            const uint32_t gu = grid_for(std::max(n, half), c->sm_count);
            if (phase == 1) {
                VC_LAUNCH(VC_K_ROUND, vc::k_round<1>, gg, vc::RED_BLOCK, 0, st, type, in1, in2, c->d_P, tab, Vb, S, j, n, c->d_part, tr);
                VC_LAUNCH(VC_K_UPDATE, vc::k_update<1>, gu, vc::RED_BLOCK, 0, st, in1, c->d_P, tab, out, S, j, n, half);
            } else {
                VC_LAUNCH(VC_K_ROUND, vc::k_round<2>, gg, vc::RED_BLOCK, 0, st, type, in1, in2, c->d_P, tab, Vb, S, j, n, c->d_part, tr);
                VC_LAUNCH(VC_K_UPDATE, vc::k_update<2>, gu, vc::RED_BLOCK, 0, st, in2, c->d_P, tab, out, S, j, n, half);
            }
            tab = out;
            tr += 3;
        }
    }
    const uint32_t used = std::min<uint32_t>(s, vc::LINE_NT + vc::LINE_TB);
    VC_LAUNCH(VC_K_LINE, vc::k_line, 1u << (s - used), 256, vc::line_smem_words(s) * 8, st, Vb, s, S, c->d_part, tr);
    return cudaGetLastError() == cudaSuccess ? VC_OK : VC_ERR_CUDA;
}

extern "C" int vc_prove_layer(vc_circuit *c, uint32_t layer, uint64_t seed, uint64_t *d_transcript, uint64_t cap_words,
                              void *cuda_stream) {
    if (!c || !d_transcript) return VC_ERR_ARG;
    if (layer >= c->d) return VC_ERR_ARG;
    if (c->next_layer < 0 || (uint32_t)c->next_layer != layer) return VC_ERR_STATE;
    if (layer > 0 && seed != c->seed) return VC_ERR_STATE;
    if (cap_words < c->layer_words(layer)) return VC_ERR_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int rc;
    if (c->hosted) rc = vc::hosted_prove_layer(c, layer, seed, d_transcript, st);
    else if (layer == 0 && c->sum_out) rc = vc::enqueue_sum_layer(c, seed, d_transcript, st);
    else if (c->schedule != 1 && vc::fused_supported(c, layer)) rc = vc::enqueue_layer_fused(c, layer, seed, d_transcript, st);
    else rc = vc::enqueue_layer_streaming(c, layer, seed, d_transcript, st);
    if (rc != VC_OK) return rc;
    c->seed = seed;
    c->next_layer = (int)layer + 1;
    return VC_OK;
}

extern "C" int vc_prove(vc_circuit *c, uint64_t seed, uint64_t *d_transcript, uint64_t cap_words, void *cuda_stream) {
    if (!c || !d_transcript) return VC_ERR_ARG;
    if (cap_words < c->total_words) return VC_ERR_ARG;
    if (c->next_layer != 0) return VC_ERR_STATE;
    if (!c->hosted && c->schedule != 1 && vc::fused_supported(c, 0)) {     // whole proof in one cooperative launch
        int rc = VC_OK;
        if (c->sum_out) rc = vc::enqueue_sum_layer(c, seed, d_transcript, (cudaStream_t)cuda_stream);   // then the fan-in-two layers 1 .. d-1
        if (rc == VC_OK && c->first_pair_layer() < c->d)
            rc = vc::enqueue_layers_fused(c, c->first_pair_layer(), c->d, seed, d_transcript + (c->sum_out ? c->layer_words(0) : 0), (cudaStream_t)cuda_stream);
        if (rc != VC_OK) return rc;
        c->seed = seed;
        c->next_layer = (int)c->d;
        return VC_OK;
    }
    uint64_t w = 0;
    for (uint32_t i = 0; i < c->d; i++) {
        const uint64_t nw = c->layer_words(i);
        int rc = vc_prove_layer(c, i, seed, d_transcript + w, nw, cuda_stream);
        if (rc != VC_OK) return rc;
        w += nw;
    }
    return VC_OK;
}

extern "C" int vc_run_host(vc_circuit *c, const uint64_t *h_input, uint64_t seed, uint64_t *h_outputs,
                           uint64_t *h_transcript, uint64_t cap_words, void *cuda_stream) {
    if (!c || !h_input || !h_outputs || !h_transcript) return VC_ERR_ARG;
    if (cap_words < c->total_words) return VC_ERR_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t n_in = (size_t)1 << c->log_input, n_out = (size_t)1 << c->logs[0];
    // H2D straight into the handle's own input table V_d; vc_evaluate then checks it in place
    CUDA_TRY(cudaMemcpyAsync(c->d_V[c->d], h_input, n_in * 8, cudaMemcpyHostToDevice, st));
    int rc = vc_evaluate(c, c->d_V[c->d], nullptr, cuda_stream);
    if (rc == VC_OK) rc = vc_prove(c, seed, c->d_tr, c->total_words, cuda_stream);
    if (rc != VC_OK) return rc;
    CUDA_TRY(cudaMemcpyAsync(h_outputs, c->d_V[0], n_out * 8, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaMemcpyAsync(h_transcript, c->d_tr, c->total_words * 8, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    uint32_t flags = 0;
    CUDA_TRY(cudaMemcpy(&flags, &c->d_state->flags, 4, cudaMemcpyDeviceToHost));
    return (flags & 1u) ? VC_ERR_ARG : VC_OK;
}

// ------------------------------------------------------------------ sizes, debug, probes
extern "C" uint64_t vc_transcript_words(const vc_circuit *c, uint32_t layer) {
    return (c && layer < c->d) ? c->layer_words(layer) : 0;
}
extern "C" uint64_t vc_total_transcript_words(const vc_circuit *c) { return c ? c->total_words : 0; }
extern "C" uint32_t vc_depth(const vc_circuit *c) { return c ? c->d : 0; }
extern "C" uint32_t vc_log_size(const vc_circuit *c, uint32_t layer) { return (c && layer <= c->d) ? c->logs[layer] : 0; }
extern "C" uint64_t vc_launch_count(void) { return vc::g_launches.load(); }

extern "C" int vc_set_schedule(vc_circuit *c, int schedule) {
    if (!c || schedule < 0 || schedule > 2) return VC_ERR_ARG;
    if ((schedule == 2) != c->hosted) return VC_ERR_STATE;      // schedule 2 is the one schedule of a hosted circuit, and only of it
    c->schedule = schedule;
    return VC_OK;
}

extern "C" int vc_debug_state(const vc_circuit *c, uint64_t *h_z64, uint64_t *h_claim, uint64_t *h_ctr, void *cuda_stream) {
    if (!c) return VC_ERR_ARG;
    CUDA_TRY(cudaStreamSynchronize((cudaStream_t)cuda_stream));
    vc::DevState hs;
    CUDA_TRY(cudaMemcpy(&hs, c->d_state, sizeof(hs), cudaMemcpyDeviceToHost));
    if (h_z64) std::memcpy(h_z64, hs.z, sizeof(hs.z));
    if (h_claim) *h_claim = hs.claim;
    if (h_ctr) *h_ctr = hs.ctr;
    return VC_OK;
}

extern "C" int vc_debug_values(const vc_circuit *c, uint32_t layer, uint64_t *h_values, void *cuda_stream) {
    if (!c || !h_values || layer > c->d) return VC_ERR_ARG;
    CUDA_TRY(cudaStreamSynchronize((cudaStream_t)cuda_stream));
    CUDA_TRY(cudaMemcpy(h_values, c->d_V[layer], (size_t)8 << c->logs[layer], cudaMemcpyDeviceToHost));
    return VC_OK;
}

extern "C" int vc_debug_layer_stamps(const vc_circuit *c, uint64_t *h_ns, void *cuda_stream) {
    if (!c || !h_ns) return VC_ERR_ARG;
    return vc::fused_stamps(c, h_ns, (cudaStream_t)cuda_stream);
}

extern "C" int vc_debug_layer_kinds(const vc_circuit *c, uint32_t *h_kind) {
    if (!c || !h_kind) return VC_ERR_ARG;
    return vc::fused_layer_kinds(c, h_kind);
}

extern "C" int vc_debug_layer_wiring(const vc_circuit *c, uint32_t *h_mode) {
    if (!c || !h_mode) return VC_ERR_ARG;
    for (uint32_t i = 0; i < c->d; i++) h_mode[i] = c->wiring[i];
    return VC_OK;
}

extern "C" int vc_debug_trace(const vc_circuit *c, uint64_t *h_words, uint32_t n_words, void *cuda_stream) {
    if (!c || !h_words) return VC_ERR_ARG;
    return vc::fused_trace(c, h_words, n_words, (cudaStream_t)cuda_stream);
}

extern "C" int vc_status(const vc_circuit *c, uint32_t *h_flags, void *cuda_stream) {
    if (!c || !h_flags) return VC_ERR_ARG;
    CUDA_TRY(cudaStreamSynchronize((cudaStream_t)cuda_stream));
    CUDA_TRY(cudaMemcpy(h_flags, &c->d_state->flags, 4, cudaMemcpyDeviceToHost));
    return VC_OK;
}

namespace vc {
__global__ void k_fieldop(int op, const uint64_t *a, const uint64_t *b, uint64_t *out, uint64_t n) {
    for (uint64_t i = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x) {
        uint64_t x = a[i], y = b[i], r;
        if (op == 0) r = fp61::add(x, y);
        else if (op == 1) r = fp61::sub(x, y);
        else if (op == 2) r = fp61::mul(x, y);
        else if (op == 3) r = fp61::draw(x, y);
        else { acc128 acc; acc.clear(); for (int k = 0; k < 64; k++) acc.mac(x, y); r = acc.value(); }  // 64 x*y, lazily
        out[i] = r;
    }
}
// ILP independent dependent-chains of fp61 multiplies per thread: the integer-multiply roofline probe
template <int ILP>
__global__ void k_bench_modmul(uint32_t iters, uint64_t *out) {
    uint64_t x[ILP];
    const uint64_t tid = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x;
#pragma unroll
    for (int k = 0; k < ILP; k++) x[k] = fp61::draw(tid, k) | 1;
    const uint64_t m = fp61::draw(12345, tid);
    for (uint32_t i = 0; i < iters; i++) {
#pragma unroll
        for (int k = 0; k < ILP; k++) x[k] = fp61::mul(x[k], m);
    }
    uint64_t r = 0;
#pragma unroll
    for (int k = 0; k < ILP; k++) r = fp61::add(r, x[k]);
    out[tid] = r;
}
}  // namespace vc

extern "C" int vc_debug_fieldop(int op, const uint64_t *d_a, const uint64_t *d_b, uint64_t *d_out, uint64_t n,
                                void *cuda_stream) {
    if (!d_a || !d_b || !d_out || op < 0 || op > 4) return VC_ERR_ARG;
    if (n == 0) return VC_OK;
    VC_LAUNCH(VC_K_MISC, vc::k_fieldop, (uint32_t)std::min<uint64_t>((n + 255) / 256, 1184), 256, 0, (cudaStream_t)cuda_stream, op, d_a, d_b, d_out, n);
    CUDA_TRY(cudaGetLastError());
    return VC_OK;
}

extern "C" int vc_bench_modmul(uint32_t grid, uint32_t block, uint32_t iters, uint32_t ilp, uint64_t *d_out, void *cuda_stream) {
    if (!d_out || grid == 0 || block == 0 || block > 1024) return VC_ERR_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    switch (ilp) {
    case 1: VC_LAUNCH(VC_K_MISC, vc::k_bench_modmul<1>, grid, block, 0, st, iters, d_out); break;
    case 2: VC_LAUNCH(VC_K_MISC, vc::k_bench_modmul<2>, grid, block, 0, st, iters, d_out); break;
    case 4: VC_LAUNCH(VC_K_MISC, vc::k_bench_modmul<4>, grid, block, 0, st, iters, d_out); break;
    case 8: VC_LAUNCH(VC_K_MISC, vc::k_bench_modmul<8>, grid, block, 0, st, iters, d_out); break;
    default: return VC_ERR_ARG;
    }
    CUDA_TRY(cudaGetLastError());
    return VC_OK;
}

// ------------------------------------------------------------------ per-kernel-kind timing for bench.py's roofline
extern "C" int vc_profile_enable(int on) {
    std::lock_guard<std::mutex> lk(vc::g_registry_mutex);
    for (auto &r : vc::g_prof) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
    vc::g_prof.clear();
    vc::g_profile = on != 0;
    return VC_OK;
}
extern "C" int vc_profile_read(uint64_t *launches, double *ms) {
    if (!launches || !ms) return VC_ERR_ARG;
    CUDA_TRY(cudaDeviceSynchronize());
    std::lock_guard<std::mutex> lk(vc::g_registry_mutex);
    for (int k = 0; k < VC_K_COUNT; k++) { launches[k] = 0; ms[k] = 0.0; }
    for (auto &r : vc::g_prof) {
        float t = 0.f;
        CUDA_TRY(cudaEventElapsedTime(&t, r.a, r.b));
        launches[r.kind] += 1; ms[r.kind] += t;
        cudaEventDestroy(r.a); cudaEventDestroy(r.b);
    }
    vc::g_prof.clear();
    return VC_OK;
}
