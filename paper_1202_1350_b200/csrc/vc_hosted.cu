// vc_hosted.cu — SURVEY.md §8(f) NEXT-3: the "copy-every-message approach" (§5.1.3), the paper's stated
// future work, for layers whose gates do not fit device memory.
//
// "copy part of a layer at a time from the host to the device, and compute the contribution of each gate in
// the part to the prover's message before swapping the part back to host memory and bringing in the next part ... for each
// message j, the entirety of the ith layer must be loaded piece-by-piece into device memory."
//
// A circuit loaded with vc_circuit_load_hosted keeps its per-gate data — the records (type, in1, in2: 9 B per gate) and the
// weights P[g] (8 B per gate) — in PINNED HOST memory.  The device holds the value tables V_i (8 B per gate; the round
// kernel gathers from V_{i+1} at random), the two fold tables and two chunk slots of 2^chunk_log gates.  Every message
// streams the whole layer through the slots:
//
//     copy-in stream   H2D  records (+ weights) of chunk k+1            |  overlapped
//     caller's stream  k_cem_round on chunk k                           |  (events per slot)
//     copy-out stream  D2H  weights of chunk k-1 back to the host       |
//
// Two ways to have the weights P[g] = beta(z, g) x (chi factors of the challenges so far) at hand (vc_hosted_set_weights):
//   recompute (default): the kernel forms P[g] from the record alone - beta by direct product over the bits of g, the chi
//       factors over the bound bits of in1 (and in2) - up to ~60 multiplies per gate and message, cheap next to 9 B per
//       gate over the host link, so nothing but the records ever crosses the link: 9 B per gate and message, one direction;
//   swap (the paper's wording: "swapping each piece back to host memory"): the weights live in a pinned host
//       array; a piece brings its weights along (8 B per gate up), the kernel applies the pending update of the previous
//       challenge (it exists only once every piece of the previous message has been reduced) before the gate's
//       contribution, and the updated weights travel back on the copy-out stream (8 B per gate down): 25 B per gate and message.
// A layer that fits ONE slot is copied once and stays there for all of its messages, weights included: the paper's
// "copy-once-per-layer approach" (§5.1.2); only wider layers are streamed per message.
// Round 0 of a layer computes beta either way (a3) and, for layer 0, the start claim.  The message of a round is the sum over
// pieces of the per-piece sums (a device accumulator; the kernel of the last piece writes the message and draws the
// challenge).  Fold tables, line restriction and the sum gate are the resident kernels of the streaming schedule.  Results
// are bit-identical to the resident schedules (tests/test_gpu_hosted.py compares with the oracle, both ways).
#include <cuda_runtime.h>

#include <algorithm>
#include <cstring>

#include "vc_circuit.hpp"
#include "vc_kernels.cuh"
#include "vc_line.cuh"
#include "vc_round.cuh"

namespace vc {

static inline uint32_t grid_for(uint64_t n, int sm_count, int per_thread = 4) {
    uint64_t b = (n + (uint64_t)RED_BLOCK * per_thread - 1) / ((uint64_t)RED_BLOCK * per_thread);
    const uint64_t cap = (uint64_t)sm_count * 4;
    return (uint32_t)std::min<uint64_t>(std::max<uint64_t>(b, 1), cap);
}

#define H_TRY(x) do { if ((x) != cudaSuccess) { (void)cudaGetLastError(); return VC_ERR_CUDA; } } while (0)

// One chunk of one message.  mode 0: first round of the layer, P[g] = beta(z, g0 + g) computed here (and, for layer 0, the
// start claim sum beta V_0); mode 1: a later round of the same phase; mode 2: first round of phase 2.  `last`: this chunk
// completes the message.  recompute != 0: P from the record (beta and the chi factors of r1[0..), r2[0..)); else P comes in
// Pw, gets the pending factor of the previous challenge (bit j-1 of this phase's index; bit s-1 of in1 in mode 2) and goes
// back through Pw.
template <int PHASE>
__global__ void __launch_bounds__(RED_BLOCK)
k_cem_round(const uint8_t *__restrict__ type, const uint32_t *__restrict__ in1, const uint32_t *__restrict__ in2, uint64_t *__restrict__ Pw,
            uint32_t g0, uint32_t cnt, uint32_t si, const uint64_t *__restrict__ Vi, const uint64_t *__restrict__ tab,
            const uint64_t *__restrict__ Vb, DevState *st, uint32_t j, uint32_t s, int mode, int last, int set_claim, int recompute,
            uint64_t *part, uint64_t *acc, uint64_t *tr) {
    __shared__ uint64_t red[4 * 32];
    __shared__ uint64_t zs[MAX_VARS], r1s[MAX_VARS], r2s[MAX_VARS];
    if (threadIdx.x < MAX_VARS) { zs[threadIdx.x] = st->z[threadIdx.x]; r1s[threadIdx.x] = st->r1[threadIdx.x]; r2s[threadIdx.x] = st->r2[threadIdx.x]; }
    __syncthreads();
    acc128 a0, a1, a2, a3; a0.clear(); a1.clear(); a2.clear(); a3.clear();
    uint64_t s0 = 0, s1 = 0, s2 = 0, s3 = 0; int it = 0;
    const uint64_t v1 = PHASE == 2 ? st->v1 : 0;
    const uint64_t rp = st->r, omrp = fp61::sub(1, rp);
    const uint32_t n1 = PHASE == 1 ? j : s, n2 = PHASE == 1 ? 0u : j;    // bound bits of in1 / in2 when this message is formed
    for (uint32_t g = blockIdx.x * blockDim.x + threadIdx.x; g < cnt; g += gridDim.x * blockDim.x) {
        const uint32_t t = type[g], i1 = in1[g], i2 = in2[g];
        uint64_t P;
        if (mode == 0 || recompute) {
            const uint32_t gg = g0 + g;
            P = 1;
            for (uint32_t k = 0; k < si; k++) P = fp61::mul(P, fp61::chi((gg >> k) & 1u, zs[k]));
            if (mode == 0 && set_claim) a3.mac(P, Vi[gg]);
            if (mode != 0) {
                uint64_t e1 = 1, e2 = 1;                                 // two more chains, independent of the first
                for (uint32_t k = 0; k < n1; k++) e1 = fp61::mul(e1, fp61::chi((i1 >> k) & 1u, r1s[k]));
                for (uint32_t k = 0; k != n2; k++) e2 = fp61::mul(e2, fp61::chi((i2 >> k) & 1u, r2s[k]));
                P = fp61::mul(P, fp61::mul(e1, e2));
            }
        } else {
            const uint32_t pb = mode == 1 ? (((PHASE == 1 ? i1 : i2) >> (j - 1)) & 1u) : ((i1 >> (s - 1)) & 1u);
            P = fp61::mul(Pw[g], pb ? rp : omrp);
        }
        if (!recompute) Pw[g] = P;
        const uint32_t idx = PHASE == 1 ? i1 : i2;
        const uint32_t b = (idx >> j) & 1u, u = idx >> (j + 1);
        const ulonglong2 pr = *reinterpret_cast<const ulonglong2 *>(tab + 2 * (size_t)u);
        const uint64_t other = PHASE == 1 ? Vb[i2] : v1;
        gate_terms<PHASE>(t, P, other, b, pr.x, pr.y, a0, a1, a2);
        if (++it == 32) {
            s0 = fp61::add(s0, a0.value()); s1 = fp61::add(s1, a1.value()); s2 = fp61::add(s2, a2.value()); s3 = fp61::add(s3, a3.value());
            a0.clear(); a1.clear(); a2.clear(); a3.clear(); it = 0;
        }
    }
    uint64_t v[4] = {fp61::add(s0, a0.value()), fp61::add(s1, a1.value()), fp61::add(s2, a2.value()), fp61::add(s3, a3.value())};
    if (grid_sum_last_block<4>(v, part, st, red) && threadIdx.x == 0) {
#pragma unroll
        for (int k = 0; k < 4; k++) v[k] = fp61::add(acc[k], v[k]);
        if (!last) {
#pragma unroll
            for (int k = 0; k < 4; k++) acc[k] = v[k];
        } else {
            tr[0] = v[0]; tr[1] = v[1]; tr[2] = v[2];
            st->G[0] = v[0]; st->G[1] = v[1]; st->G[2] = v[2];
            if (set_claim) st->claim = v[3];
            const uint64_t r = fp61::draw(st->seed, st->ctr);      // only now: every chunk of this message is in
            st->ctr += 1;
            st->r = r;
            if (PHASE == 1) st->r1[j] = r; else st->r2[j] = r;
            acc[0] = 0; acc[1] = 0; acc[2] = 0; acc[3] = 0;
        }
    }
}

// ------------------------------------------------------------------ host side
int hosted_init(vc_circuit *c) {
    const size_t ch = (size_t)1 << c->chunk_log;
    // pin the records where they are (no second host copy).  Small arrays stay pageable: two of them can share a page, which
    // cudaHostRegister refuses, and their copies are staged by the driver in stream order all the same.
    auto pin = [&](void *p, size_t bytes) {
        if (bytes < (1u << 16)) return;
        if (cudaHostRegister(p, bytes, cudaHostRegisterDefault) == cudaSuccess) c->pinned_ptrs.push_back(p);
        else (void)cudaGetLastError();
    };
    for (uint32_t i = 0; i < c->d; i++) {
        pin(c->h_type[i].data(), c->h_type[i].size());
        pin(c->h_in1[i].data(), c->h_in1[i].size() * 4);
        pin(c->h_in2[i].data(), c->h_in2[i].size() * 4);
    }
    uint64_t max_gates = 1;
    for (uint32_t i = 0; i < c->d; i++) max_gates = std::max<uint64_t>(max_gates, 1ull << c->logs[i]);
    if (cudaMallocHost(&c->p_P, max_gates * 8) != cudaSuccess) { (void)cudaGetLastError(); return VC_ERR_NOMEM; }
    for (auto &sl : c->slot) {
        if (cudaMalloc(&sl.type, ch) != cudaSuccess || cudaMalloc(&sl.in1, ch * 4) != cudaSuccess || cudaMalloc(&sl.in2, ch * 4) != cudaSuccess ||
            cudaMalloc(&sl.P, ch * 8) != cudaSuccess) { (void)cudaGetLastError(); return VC_ERR_NOMEM; }
        H_TRY(cudaEventCreateWithFlags(&sl.ready, cudaEventDisableTiming));
        H_TRY(cudaEventCreateWithFlags(&sl.done, cudaEventDisableTiming));
        H_TRY(cudaEventCreateWithFlags(&sl.back, cudaEventDisableTiming));
    }
    H_TRY(cudaStreamCreateWithFlags(&c->s_in, cudaStreamNonBlocking));
    H_TRY(cudaStreamCreateWithFlags(&c->s_out, cudaStreamNonBlocking));
    H_TRY(cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming));
    H_TRY(cudaEventCreateWithFlags(&c->ev_round, cudaEventDisableTiming));
    if (cudaMalloc(&c->d_acc, 4 * 8) != cudaSuccess) { (void)cudaGetLastError(); return VC_ERR_NOMEM; }
    H_TRY(cudaMemset(c->d_acc, 0, 4 * 8));
    H_TRY(cudaFuncSetAttribute(k_line, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 1024));
    return VC_OK;
}

void hosted_free(vc_circuit *c) {
    if (!c->hosted) return;
    if (c->s_in) { cudaStreamSynchronize(c->s_in); cudaStreamDestroy(c->s_in); }
    if (c->s_out) { cudaStreamSynchronize(c->s_out); cudaStreamDestroy(c->s_out); }
    for (void *p : c->pinned_ptrs) cudaHostUnregister(p);
    c->pinned_ptrs.clear();
    cudaFreeHost(c->p_P);
    for (auto &sl : c->slot) {
        cudaFree(sl.type); cudaFree(sl.in1); cudaFree(sl.in2); cudaFree(sl.P);
        if (sl.ready) cudaEventDestroy(sl.ready);
        if (sl.done) cudaEventDestroy(sl.done);
        if (sl.back) cudaEventDestroy(sl.back);
    }
    if (c->ev_fork) cudaEventDestroy(c->ev_fork);
    if (c->ev_round) cudaEventDestroy(c->ev_round);
    cudaFree(c->d_acc);
    (void)cudaGetLastError();
}

// the copy streams join the caller's stream: nothing they do starts before the work already enqueued on st
static int fork_streams(vc_circuit *c, cudaStream_t st) {
    H_TRY(cudaEventRecord(c->ev_fork, st));
    H_TRY(cudaStreamWaitEvent(c->s_in, c->ev_fork, 0));
    H_TRY(cudaStreamWaitEvent(c->s_out, c->ev_fork, 0));
    return VC_OK;
}
// ... and the caller's stream waits for the last copy-out before anything enqueued after this call
static int join_streams(vc_circuit *c, cudaStream_t st) {
    H_TRY(cudaEventRecord(c->ev_round, c->s_out));
    H_TRY(cudaStreamWaitEvent(st, c->ev_round, 0));
    H_TRY(cudaEventRecord(c->ev_fork, c->s_in));
    H_TRY(cudaStreamWaitEvent(st, c->ev_fork, 0));
    return VC_OK;
}

// H2D of one chunk's records (and weights) into its slot, ordered after the slot's previous use
static int chunk_in(vc_circuit *c, uint32_t layer, uint32_t k, uint32_t g0, uint32_t cnt, bool with_P) {
    auto &sl = c->slot[k & 1];
    H_TRY(cudaStreamWaitEvent(c->s_in, sl.done, 0));
    H_TRY(cudaStreamWaitEvent(c->s_in, sl.back, 0));
    H_TRY(cudaMemcpyAsync(sl.type, c->h_type[layer].data() + g0, cnt, cudaMemcpyHostToDevice, c->s_in));
    H_TRY(cudaMemcpyAsync(sl.in1, c->h_in1[layer].data() + g0, (size_t)cnt * 4, cudaMemcpyHostToDevice, c->s_in));
    H_TRY(cudaMemcpyAsync(sl.in2, c->h_in2[layer].data() + g0, (size_t)cnt * 4, cudaMemcpyHostToDevice, c->s_in));
    c->h2d_bytes += (uint64_t)cnt * 9;
    if (with_P) { H_TRY(cudaMemcpyAsync(sl.P, c->p_P + g0, (size_t)cnt * 8, cudaMemcpyHostToDevice, c->s_in)); c->h2d_bytes += (uint64_t)cnt * 8; }
    H_TRY(cudaEventRecord(sl.ready, c->s_in));
    return VC_OK;
}

int hosted_evaluate(vc_circuit *c, const uint64_t *d_input, uint64_t *d_outputs, cudaStream_t st) {
    const uint32_t d = c->d;
    const uint64_t n_in = 1ull << c->log_input;
    c->h2d_bytes = 0; c->d2h_bytes = 0;
    VC_LAUNCH(VC_K_EVAL, k_copy_input, grid_for(n_in, c->sm_count), RED_BLOCK, 0, st, d_input, c->d_V[d], n_in, c->d_state);
    int rc = fork_streams(c, st);
    if (rc != VC_OK) return rc;
    const uint32_t ch = 1u << c->chunk_log;
    uint32_t k = 0;
    for (int i = (int)d - 1; i >= (int)c->first_pair_layer(); i--) {
        const uint32_t n = 1u << c->logs[i];
        for (uint32_t g0 = 0; g0 < n; g0 += ch, k++) {
            const uint32_t cnt = std::min(ch, n - g0);
            auto &sl = c->slot[k & 1];
            if ((rc = chunk_in(c, (uint32_t)i, k, g0, cnt, false)) != VC_OK) return rc;
            H_TRY(cudaStreamWaitEvent(st, sl.ready, 0));
            VC_LAUNCH(VC_K_EVAL, k_eval, grid_for(cnt, c->sm_count, 2), RED_BLOCK, 0, st, sl.type, sl.in1, sl.in2, c->d_V[i + 1], c->d_V[i] + g0,
                      (i == 0 && d_outputs ? d_outputs + g0 : (uint64_t *)nullptr), cnt);
            H_TRY(cudaEventRecord(sl.done, st));
        }
    }
    H_TRY(cudaGetLastError());
    if (c->sum_out && (rc = enqueue_sum_eval(c, d_outputs, st)) != VC_OK) return rc;
    return join_streams(c, st);
}

int hosted_prove_layer(vc_circuit *c, uint32_t layer, uint64_t seed, uint64_t *d_tr, cudaStream_t st) {
    if (layer == 0) { c->h2d_bytes = 0; c->d2h_bytes = 0; }
    if (layer == 0 && c->sum_out) return enqueue_sum_layer(c, seed, d_tr, st);     // tables only: nothing to stream
    const uint32_t si = c->logs[layer], s = c->logs[layer + 1];
    const uint32_t n = 1u << si, ch = 1u << c->chunk_log;
    const uint32_t nchunks = (n + ch - 1) / ch;
    DevState *S = c->d_state;
    const uint64_t *Vb = c->d_V[layer + 1];
    if (layer == 0) VC_LAUNCH(VC_K_SETUP, k_start, 1, 64, 0, st, S, seed, si);
    H_TRY(cudaMemsetAsync(c->d_acc, 0, 4 * 8, st));
    int rc = fork_streams(c, st);
    if (rc != VC_OK) return rc;
    uint64_t *tr = d_tr;
    uint32_t k = 0;
    // A layer that fits one slot is copied ONCE and stays there, weights included, for all of its messages: the paper's
    // "copy-once-per-layer approach" (§5.1.2, the one its experiments used); only wider layers pay per message.
    const bool once = nchunks == 1;
    for (int phase = 1; phase <= 2; phase++) {
        const uint64_t *tab = Vb;
        for (uint32_t j = 0; j < s; j++) {
            const int mode = (phase == 1 && j == 0) ? 0 : ((phase == 2 && j == 0) ? 2 : 1);
            const bool swap = c->hosted_swap && !once;
            if (swap && mode != 0) H_TRY(cudaStreamWaitEvent(c->s_in, c->ev_round, 0));  // the weights of the previous message are back on the host
            for (uint32_t q = 0; q < nchunks; q++, k++) {
                const uint32_t g0 = q * ch, cnt = std::min(ch, n - g0);
                auto &sl = c->slot[once ? 0 : (k & 1)];
                if (!once || mode == 0) {
                    if ((rc = chunk_in(c, layer, once ? 0 : k, g0, cnt, swap && mode != 0)) != VC_OK) return rc;
                    H_TRY(cudaStreamWaitEvent(st, sl.ready, 0));
                }
                const int last = q + 1 == nchunks, set_claim = layer == 0 && mode == 0;
                const int recompute = (swap || once) ? 0 : 1;        // once: the weights stay in the slot between messages
                const uint32_t gg = grid_for(cnt, c->sm_count);
                if (phase == 1)
                    VC_LAUNCH(VC_K_ROUND, k_cem_round<1>, gg, RED_BLOCK, 0, st, sl.type, sl.in1, sl.in2, sl.P, g0, cnt, si, c->d_V[layer], tab, Vb, S, j, s,
                              mode, last, set_claim, recompute, c->d_part, c->d_acc, tr);
                else
                    VC_LAUNCH(VC_K_ROUND, k_cem_round<2>, gg, RED_BLOCK, 0, st, sl.type, sl.in1, sl.in2, sl.P, g0, cnt, si, c->d_V[layer], tab, Vb, S, j, s,
                              mode, last, set_claim, recompute, c->d_part, c->d_acc, tr);
                H_TRY(cudaEventRecord(sl.done, st));
                if (swap) {                                                              // swap the piece back
                    H_TRY(cudaStreamWaitEvent(c->s_out, sl.done, 0));
                    H_TRY(cudaMemcpyAsync(c->p_P + g0, sl.P, (size_t)cnt * 8, cudaMemcpyDeviceToHost, c->s_out));
                    c->d2h_bytes += (uint64_t)cnt * 8;
                    H_TRY(cudaEventRecord(sl.back, c->s_out));
                }
            }
            if (swap) H_TRY(cudaEventRecord(c->ev_round, c->s_out));
            // a6, the table half: fold by the challenge the last chunk's kernel drew (no gates in this launch)
            uint64_t *out = (j & 1) ? c->d_T1 : c->d_T0;
            const uint32_t half = 1u << (s - j - 1);
            if (phase == 1)
                VC_LAUNCH(VC_K_UPDATE, k_update<1>, grid_for(half, c->sm_count), RED_BLOCK, 0, st, (const uint32_t *)nullptr, (uint64_t *)nullptr, tab, out, S, j, 0u, half);
            else
                VC_LAUNCH(VC_K_UPDATE, k_update<2>, grid_for(half, c->sm_count), RED_BLOCK, 0, st, (const uint32_t *)nullptr, (uint64_t *)nullptr, tab, out, S, j, 0u, half);
            tab = out;
            tr += 3;
        }
    }
    const uint32_t used = std::min<uint32_t>(s, LINE_NT + LINE_TB);
    VC_LAUNCH(VC_K_LINE, k_line, 1u << (s - used), 256, line_smem_words(s) * 8, st, Vb, s, S, c->d_part, tr);
    H_TRY(cudaGetLastError());
    return join_streams(c, st);
}

}  // namespace vc
