// vc_circuit.hpp — the opaque handle behind include/vc.h (host side).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>
#include <mutex>
#include <vector>

#include "../../include/vc.h"
#include "vc_state.cuh"

struct vc_circuit {
    uint32_t d = 0, log_input = 0;
    std::vector<uint32_t> logs;                 // logs[i] = log2 size of layer i, i = 0..d (d = input)
    // host copies of the records (the verifier runs on the host)
    std::vector<std::vector<uint8_t>> h_type;
    std::vector<std::vector<uint32_t>> h_in1, h_in2;
    // device: records (SoA), value tables
    std::vector<uint8_t *> d_type;
    std::vector<uint32_t *> d_in1, d_in2;
    std::vector<uint64_t *> d_V;                // d+1 tables, V[d] = input copy
    // per-layer wiring class (set at load): 1 = tree (in1 = 2g, in2 = 2g+1), 2 = self (in1 = in2 = g), both with a single
    // gate type; 3 = bit-field rule (wrule[i]); else 0 = generic (records are read)
    std::vector<uint32_t> wiring;
    std::vector<vc::WireRule> wrule;
    // scratch
    uint64_t *d_P = nullptr;                    // weights, max layer size
    uint64_t *d_T0 = nullptr, *d_T1 = nullptr;  // fold ping-pong
    uint64_t *d_part = nullptr;                 // block partials
    uint64_t *d_tr = nullptr;                   // internal transcript buffer (vc_run_host)
    vc::DevState *d_state = nullptr;
    size_t part_words = 0;
    uint64_t total_words = 0;
    // proof sequencing
    int next_layer = -1;                        // -1: vc_evaluate not called yet
    uint64_t seed = 0;
    int schedule = 0;
    int sm_count = 148;
    int coop_ok = 0;

    // hosted circuits (vc_circuit_load_hosted; vc_hosted.cu): records and weights stay in pinned host memory and are streamed
    // through two device slots for every message (the copy-every-message approach)
    bool hosted = false;
    uint32_t chunk_log = 0;
    bool hosted_swap = false;                   // weights swapped through host memory (the paper's wording) instead of recomputed per message
    std::vector<void *> pinned_ptrs;            // record arrays registered with cudaHostRegister
    uint64_t *p_P = nullptr;                    // pinned host weights, max layer size
    struct HostedSlot { uint8_t *type; uint32_t *in1, *in2; uint64_t *P; cudaEvent_t ready, done, back; };
    HostedSlot slot[2] = {};
    cudaStream_t s_in = nullptr, s_out = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_round = nullptr;
    uint64_t *d_acc = nullptr;                  // running sums of a message across chunks (+ the start claim)
    uint64_t h2d_bytes = 0, d2h_bytes = 0;      // moved by the last evaluation / proof of a hosted circuit
    bool sum_out = false;                       // layer 0 is the single VC_SUM gate over all of layer 1

    uint32_t log_below(uint32_t i) const { return logs[i + 1]; }
    // transcript words of layer i: 2s x (G0,G1,G2) then q[0..s]; the sum gate: s x (G0,G1)
    uint64_t layer_words(uint32_t i) const { return (sum_out && i == 0) ? 2ull * logs[1] : 7ull * logs[i + 1] + 1; }
    uint32_t first_pair_layer() const { return sum_out ? 1u : 0u; }   // first layer proved by the fan-in-two engines
};

namespace vc {
extern std::atomic<uint64_t> g_launches;
extern std::mutex g_registry_mutex;         // guards the process-wide registries (fused plans, verifier scratch, profile records)
struct ProfRec { int kind; cudaEvent_t a, b; };
extern bool g_profile;                      // vc_profile_enable: CUDA events around every launch, by kind
void prof_push(int kind, cudaEvent_t a, cudaEvent_t b);
int enqueue_layer_streaming(vc_circuit *c, uint32_t layer, uint64_t seed, uint64_t *d_tr, cudaStream_t st);
int enqueue_sum_layer(vc_circuit *c, uint64_t seed, uint64_t *d_tr, cudaStream_t st);                  // vc_api.cu (vc_sum.cuh)
int enqueue_sum_eval(vc_circuit *c, uint64_t *d_outputs, cudaStream_t st);
int hosted_init(vc_circuit *c);                                                                       // vc_hosted.cu
void hosted_free(vc_circuit *c);
int hosted_evaluate(vc_circuit *c, const uint64_t *d_input, uint64_t *d_outputs, cudaStream_t st);
int hosted_prove_layer(vc_circuit *c, uint32_t layer, uint64_t seed, uint64_t *d_tr, cudaStream_t st);
int enqueue_layer_fused(vc_circuit *c, uint32_t layer, uint64_t seed, uint64_t *d_tr, cudaStream_t st);  // vc_fused.cu
int fused_supported(const vc_circuit *c, uint32_t layer);
int fused_init(vc_circuit *c);
void fused_free(const vc_circuit *c);
void verifier_free(const vc_circuit *c);   // vc_verify_gpu.cu
int fused_stamps(const vc_circuit *c, uint64_t *h, cudaStream_t st);
int fused_layer_kinds(const vc_circuit *c, uint32_t *h_kind);
int fused_trace(const vc_circuit *c, uint64_t *h, uint32_t n_words, cudaStream_t st);
int enqueue_eval_fused(vc_circuit *c, const uint64_t *d_input, uint64_t *d_outputs, cudaStream_t st);
int enqueue_layers_fused(vc_circuit *c, uint32_t begin, uint32_t end, uint64_t seed, uint64_t *d_tr, cudaStream_t st);
}  // namespace vc

// Launch + count (+ optional event pair tagged with the kernel kind, for bench.py's live roofline numbers).
#define VC_LAUNCH(kind, kern, grid, block, smem, stream, ...)                               \
    do {                                                                                    \
        cudaEvent_t ea_ = nullptr, eb_ = nullptr;                                           \
        if (vc::g_profile) { cudaEventCreate(&ea_); cudaEventCreate(&eb_); cudaEventRecord(ea_, (stream)); } \
        kern<<<(grid), (block), (smem), (stream)>>>(__VA_ARGS__);                           \
        if (vc::g_profile) { cudaEventRecord(eb_, (stream)); vc::prof_push((kind), ea_, eb_); } \
        vc::g_launches.fetch_add(1, std::memory_order_relaxed);                             \
    } while (0)
