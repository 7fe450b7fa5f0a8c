/* vc.h — C ABI of libvc.so: the GKR/CMT prover hot path over F_p, p = 2^61 - 1, on one B200.
 *
 * Protocol: PAPER.md:93-101 (§3.1, GKR iteration structure), PAPER.md:121-123 (§4.1.1, each gate
 * contributes independently to each message; contributions are reduced in F_p), PAPER.md:197 (§6.1,
 * the field).  Conventions the paper leaves open follow SURVEY.md §8(c) / DESIGN.md "Readings".
 *
 * Conventions: layer 0 = outputs, layer d = inputs; layer i has exactly 2^log_size gates; gate g of
 * layer i reads entries in1[g], in2[g] of layer i+1.  All field words are canonical uint64 in [0,p).
 * Bit k of an index is variable k (k = 0 least significant).  Challenges are H(seed, ctr++) from a
 * counter-based generator kept on the device (splitmix64 stream, low 61 bits, p -> 0).
 *
 * Every function returns an integer code (VC_OK = 0); nothing throws, aborts or prints.
 * Functions taking a `cuda_stream` (a cudaStream_t passed as void*, NULL = default stream) only
 * ENQUEUE work and return without synchronising; VC_OK then means "enqueued".
 * There is no CPU fallback: without a CUDA device every compute entry point returns VC_ERR_CUDA.
 */
#ifndef VC_H
#define VC_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct vc_circuit vc_circuit; /* opaque; owns device copies of records, V tables, scratch, proof state */

enum { VC_OK = 0, VC_ERR_ARG = 1, VC_ERR_SHAPE = 2, VC_ERR_STATE = 3, VC_ERR_CUDA = 4, VC_ERR_NOMEM = 5,
       VC_ERR_LIMIT = 6 /* a size beyond the fixed maximum of an entry point that allocates nothing */ };
enum { VC_ADD = 0, VC_MULT = 1, VC_SUB = 2, VC_RELAY = 3, VC_SUM = 4 };

/* VC_SUM — the "single sum-gate of very large fan-in at the output" (DESIGN.md
 * reading c-19).  Allowed only as the ONE gate of layer 0 (log_size 0; in1 / in2 need one placeholder entry each and are
 * not read): its in-neighbours are ALL gates of layer 1, V_0[0] = sum_w V_1[w].  Its iteration of the protocol is a
 * sum-check over the s = log_size(layer 1) variables of the multilinear extension of V_1, bit 0 first: round j emits
 * (g_j(0), g_j(1)) = the sums of the even- and odd-indexed entries of the table folded by r_0..r_{j-1}, the challenge
 * r_j is drawn on the device, and after s rounds the claim is V~_1(r) at the one point z' = r (no line restriction, no
 * tau).  Such a layer writes 2 s transcript words and takes s draws; the verifiers check g_j(0) + g_j(1) = claim and
 * continue with claim <- g_j(0) + r_j (g_j(1) - g_j(0)): fail_round = j < s, and there is no wiring check for it. */

/* One layer's gate records, structure-of-arrays, in HOST memory (copied at load; caller keeps ownership). */
typedef struct {
    uint32_t log_size;    /* the layer has exactly 2^log_size gates */
    const uint8_t *type;  /* VC_ADD L+R, VC_MULT L*R, VC_SUB L-R, VC_RELAY L; VC_SUM only as the single gate of layer 0 (above) */
    const uint32_t *in1;  /* indices into the layer below, < 2^log_size(below) */
    const uint32_t *in2;
} vc_layer;

/* vc_circuit_load — copy the circuit to the device and allocate every buffer the path needs
 * (value tables V_0..V_d, weights, fold tables, partials, proof state).  Allocation is outside any
 * timed region (scratch allocation is not counted).  "No-copying approach",
 * PAPER.md:153 (§5.1.1): the whole circuit stays resident in HBM.
 *   layers[0] = output layer ... layers[d-1] = the layer fed by the input; log_input = log2(#inputs).
 * Errors: VC_ERR_ARG (null, d = 0), VC_ERR_SHAPE (log_size > 30, a layer below of size 1, index out
 * of range, unknown type, VC_SUM anywhere but as the single gate of layer 0), VC_ERR_CUDA / VC_ERR_NOMEM. */
int vc_circuit_load(const vc_layer *layers, uint32_t d, uint32_t log_input, vc_circuit **out);

/* vc_circuit_load_hosted — the "copy-every-message approach" (§5.1.3, the paper's stated future work;
 * SURVEY.md §8(f) NEXT-3) for layers whose gates do not fit device memory.  Same arguments and checks as vc_circuit_load, but
 * the per-gate data — records (9 B per gate) and weights (8 B per gate) — stays in pinned HOST memory (the record arrays
 * are copied once into the handle and page-locked there); the device holds the value tables, the fold tables and two chunk
 * slots of 2^chunk_log gates (8 <= chunk_log <= 28, else VC_ERR_ARG).  For EVERY message of a layer the whole layer
 * is streamed through the slots piece by piece: H2D of a piece's records, the piece's contribution to the message, the
 * copies of neighbouring pieces overlapping the kernel on internal streams.  The weights are either recomputed from the
 * record for every message (default: nothing but 9 B per gate and message crosses the host link) or swapped through the
 * host array as the paper words it (vc_hosted_set_weights(c, 1): + 8 B per gate up and 8 B down per message, the pending
 * update of the previous challenge applied when the piece comes back).  A layer of at most 2^chunk_log gates is copied
 * ONCE and stays in its slot, weights included, for all of its messages (the paper's copy-once-per-layer approach,
 * PAPER.md:157 §5.1.2): only wider layers are streamed per message.  vc_evaluate streams the records once per
 * layer.  Every other call (vc_prove_layer, vc_prove, vc_run_host, vc_verify_transcript, sizes) behaves as for a resident
 * circuit and produces the same words; vc_set_schedule accepts only 2 for such a handle (and 2 only for such a handle),
 * vc_verify_transcript_device returns VC_ERR_STATE (its wiring sums need device-resident records). */
int vc_circuit_load_hosted(const vc_layer *layers, uint32_t d, uint32_t log_input, uint32_t chunk_log, vc_circuit **out);
/* hosted handles only (else VC_ERR_STATE): swap = 0 recompute the weights per message (default), 1 swap them through host
 * memory.  Takes effect at the next vc_prove_layer; set it before layer 0.  Same transcript either way. */
int vc_hosted_set_weights(vc_circuit *c, int swap);
/* bytes a hosted circuit moved over the host link in its last vc_evaluate (h2d only) or since layer 0 of its last proof;
 * VC_ERR_STATE for a resident circuit */
int vc_debug_hosted_bytes(const vc_circuit *c, uint64_t *h2d, uint64_t *d2h);

/* vc_evaluate — layered circuit evaluation (step a1; §6.2.4):
 * V_d = input; for i = d-1..0: V_i[g] = f_type(V_{i+1}[in1[g]], V_{i+1}[in2[g]])  (a VC_SUM output: the sum of V_1).
 *   d_input   DEVICE pointer, 2^log_input canonical words (read).  A word >= p is detected ON THE DEVICE while the input
 *             is copied, i.e. asynchronously: the call itself still returns VC_OK ("enqueued").  The sticky bit 0 of the
 *             status word reports it for THIS evaluation (it is cleared when vc_evaluate is enqueued): vc_status reads
 *             it after a stream synchronise, and vc_run_host, which synchronises anyway, returns VC_ERR_ARG.
 *             (SURVEY.md §8(b) "Errors": non-canonical input -> VC_ERR_ARG at load or evaluate; detection cannot be
 *             synchronous without a device round-trip inside a call that must not synchronise.)
 *   d_outputs DEVICE pointer, 2^log_size(layer 0) words (written); may be NULL.
 * Resets the proof state (next vc_prove_layer must be layer 0). */
int vc_evaluate(vc_circuit *c, const uint64_t *d_input, uint64_t *d_outputs, void *cuda_stream);

/* vc_prove_layer — one GKR iteration (steps a2-a7):
 * layer 0 first resets the challenge counter, draws z_0 and forms the start claim V~_0(z_0);
 * then beta(z,.) weights, 2*s sum-check rounds (s = log2 size of layer i+1; phase 1 binds the bits of
 * in1, phase 2 the bits of in2, LSB first; each round emits G[0],G[1],G[2] = the round polynomial at
 * t = 0,1,2, reduced mod p over all gates, then draws the challenge on the device), then the line
 * restriction q[0..s] = V~_{i+1}(r1 + t (r2 - r1)), a draw tau, z <- l(tau), claim <- q(tau).
 *   d_transcript DEVICE pointer, receives 7*s+1 words: 2s x (G0,G1,G2), then q[0..s]
 *                (a VC_SUM layer 0: 2*s words, s x (G0,G1); vc_transcript_words gives the count for any layer).
 *   cap_words    capacity of d_transcript in words (VC_ERR_ARG if < vc_transcript_words(c, layer)).
 * Must be called with layer = 0,1,...,d-1 in order after vc_evaluate, with the same seed
 * (else VC_ERR_STATE).  Leaves (z, claim, counter) on the device for the next call. */
int vc_prove_layer(vc_circuit *c, uint32_t layer, uint64_t seed, uint64_t *d_transcript, uint64_t cap_words,
                   void *cuda_stream);

/* vc_prove — convenience: vc_prove_layer for layers 0..d-1 into one device buffer (layer 0 first),
 * cap_words >= vc_total_transcript_words.  Same kernels, same order; no host round-trip. */
int vc_prove(vc_circuit *c, uint64_t seed, uint64_t *d_transcript, uint64_t cap_words, void *cuda_stream);

/* vc_run_host — the end-to-end call with HOST buffers: H2D copy of the input, vc_evaluate, vc_prove,
 * D2H copy of outputs and transcript, stream synchronised before returning.
 *   h_input 2^log_input words (read), h_outputs 2^log_size(layer 0) words (written),
 *   h_transcript cap_words words (written).  Pinned host memory makes the copies asynchronous. */
int vc_run_host(vc_circuit *c, const uint64_t *h_input, uint64_t seed, uint64_t *h_outputs,
                uint64_t *h_transcript, uint64_t cap_words, void *cuda_stream);

/* vc_verify_transcript — the verifier (PAPER.md:63-65 §2.2, :99; host code, not on the hot path).
 * Recomputes the start claim from h_outputs, checks every round (G0+G1 = claim), the wiring check
 * after 2s rounds with v1 = q[0], v2 = q[1], follows the line to the next layer, and closes with
 * claim = V~_d(z) of h_input.  All pointers HOST.  Rejection is NOT an error: returns VC_OK with
 * *accept = 0 and (fail_layer, fail_round): round m < 2s = round check m failed; round 2s = wiring
 * check failed; fail_layer = d = closing input check failed. */
int vc_verify_transcript(const vc_circuit *c, const uint64_t *h_input, const uint64_t *h_outputs, uint64_t seed,
                         const uint64_t *h_transcript, uint64_t n_words, int *accept, uint32_t *fail_layer,
                         uint32_t *fail_round);

/* vc_verify_transcript_device — the same verifier with its O(S) sums on the GPU (
 * PAPER.md:127 §4.1.2: one chi-weighted term per input element, reduced in F_p).  Three kinds of sums
 * run as kernels, all enqueued at once on cuda_stream: the start claim V~_0(z_0) of the claimed outputs, the four
 * per-type wiring sums of every layer, and the closing extension V~_d(z_d) of the input; the O(rounds) checks then run
 * on the host over the transcript (copied back: 7s+1 words per layer).  Same acceptance rule, same
 * (fail_layer, fail_round) and same error codes as vc_verify_transcript.
 *   d_input, d_outputs, d_transcript: DEVICE pointers (read); accept, fail_layer, fail_round: HOST (written).
 * Synchronises cuda_stream before returning.  Scratch for the sums is allocated on the first call for a circuit
 * (VC_ERR_NOMEM if that fails) and released by vc_circuit_free. */
int vc_verify_transcript_device(const vc_circuit *c, const uint64_t *d_input, const uint64_t *d_outputs, uint64_t seed,
                                const uint64_t *d_transcript, uint64_t n_words, int *accept, uint32_t *fail_layer,
                                uint32_t *fail_round, void *cuda_stream);

void vc_circuit_free(vc_circuit *c);
const char *vc_strerror(int code);
uint64_t vc_transcript_words(const vc_circuit *c, uint32_t layer);  /* 7*s+1; 0 if layer >= d */
uint64_t vc_total_transcript_words(const vc_circuit *c);
uint32_t vc_depth(const vc_circuit *c);
uint32_t vc_log_size(const vc_circuit *c, uint32_t layer);           /* layer = d gives log_input */

/* Debug / test helpers (synchronise the stream they are given). */
/* copies (z[0..63], claim, counter) of the proof state to the host */
int vc_debug_state(const vc_circuit *c, uint64_t *h_z64, uint64_t *h_claim, uint64_t *h_ctr, void *cuda_stream);
/* copies value table V_layer (layer = d: the input copy) to the host */
int vc_debug_values(const vc_circuit *c, uint32_t layer, uint64_t *h_values, void *cuda_stream);
/* fused schedule only: d+1 device timestamps (ns, %globaltimer): start of each layer's proof, [d] = end */
int vc_debug_layer_stamps(const vc_circuit *c, uint64_t *h_ns, void *cuda_stream);
/* fused schedule, builds with -DVC_TRACE only (all zero otherwise): the first n_words <= 65536 trace words of the last
 * launch, each (code << 48 | SM clock of CTA 0) */
int vc_debug_trace(const vc_circuit *c, uint64_t *h_words, uint32_t n_words, void *cuda_stream);
/* the device sums of the last vc_verify_transcript_device call on this circuit, n = 4 d + 2 HOST words:
 * [0] start claim, [1 + 4 i + t] wiring sum of type t of layer i, [1 + 4 d] the input extension at z_d */
int vc_debug_verifier_sums(const vc_circuit *c, uint64_t *h_sums, uint64_t n);
/* device-side status of the last vc_evaluate on this handle: 0 = fine, bit 0 = a non-canonical input word was seen */
int vc_status(const vc_circuit *c, uint32_t *h_flags, void *cuda_stream);
/* which kernel proves each layer on the fused schedule: h_kind receives d words, each one of VC_K_CLUSTER, VC_K_FUSED_NARROW,
 * VC_K_FUSED_THIN, VC_K_FUSED_WIDE (bench.py uses it to give every kernel kind its own algorithmic byte count);
 * VC_ERR_STATE when the circuit has no fused plan (streaming schedule only) */
int vc_debug_layer_kinds(const vc_circuit *c, uint32_t *h_kind);
/* vc_mle_device_noalloc — the multilinear extension of a device table at one point, for callers that cannot allocate
 * (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).  The operation is the verifier's
 * "secret" of PAPER.md:127 (§4.1.2) / :99: out = sum_u eq(u, x) V[u] over the 2^log_n words of V, every element one
 * chi-weighted term, reduced in F_p — the same arithmetic as the start-claim and closing-check kernels of
 * vc_verify_transcript_device, whose scratch is cudaMalloc'd per circuit.  Here the kernel's scratch (block partials,
 * ticket, status word) is one file-scope device array of VC_NOALLOC_SCRATCH_WORDS 64-bit words (4 KB) that every GPU
 * loading the library holds until the process exits; the call itself calls no cudaMalloc / cudaFree / allocating routine:
 * it enqueues one 16-byte memset of the scratch's ticket and status words, one kernel and one 8-byte device-to-device
 * copy on cuda_stream and returns without synchronising.
 *   d_values  DEVICE, 2^log_n words (read); a word >= p is reduced by masking to 61 bits and reported in d_out2[1]
 *   log_n     0 .. VC_NOALLOC_MAX_LOG (28: tables of up to 2^28 words = 2 GiB); larger: VC_ERR_LIMIT, nothing enqueued
 *   d_point   DEVICE, log_n canonical words x[0..log_n) (read; bit k of the index is variable k); may be NULL if log_n = 0
 *   d_out2    DEVICE, 2 words (written): [0] = the value, [1] = 1 if a word of d_values was >= p, else 0
 * The first call on a device resolves the scratch array's device address (cudaGetSymbolAddress, once per device, with that
 * device current): make one call outside any stream capture first.  All calls on a device SHARE the array: calls that
 * overlap on the GPU (different streams, several host threads) race — serialise them on one stream or with events.
 * Errors: VC_ERR_ARG (null pointer), VC_ERR_LIMIT (log_n too large), VC_ERR_CUDA. */
#define VC_NOALLOC_MAX_LOG 28
#define VC_NOALLOC_SCRATCH_WORDS 512
int vc_mle_device_noalloc(const uint64_t *d_values, uint32_t log_n, const uint64_t *d_point, uint64_t *d_out2,
                          void *cuda_stream);

/* how the prover obtains each layer's wiring (the paper's §5.1.4 computes the tree's indices instead of
 * loading them): h_mode receives d words, 0 = the stored records are read, 1 = binary tree (2g, 2g+1) computed, 2 = in1 = in2 = g
 * computed, 3 = computed from the bit-field rule vc_load fitted to the records and checked against every one of them.  The
 * records stay the definition: a layer gets a computed mode only when it reproduces all of its records. */
int vc_debug_layer_wiring(const vc_circuit *c, uint32_t *h_mode);
/* number of kernels this library has launched since load (for bench.py's gpu_launches) */
uint64_t vc_launch_count(void);
/* selects the kernel schedule: 0 = auto (default), 1 = streaming (one kernel per protocol step); 2 = copy-every-message, the
 * fixed schedule of a vc_circuit_load_hosted handle (VC_ERR_STATE for any other combination); DESIGN.md §5 (schedules 0, 1) and §9e (schedule 2) */
int vc_set_schedule(vc_circuit *c, int schedule);

/* Field/PRNG probes for the GPU unit tests: out[i] = op(a[i], b[i]) on the device, n words each,
 * all DEVICE pointers.  op: 0 add, 1 sub, 2 mul, 3 draw(seed=a[i], ctr=b[i]), 4 sum of 64 products a[i]*b[i] through the
 * lazy 128-bit accumulator (one fold at the end). */
int vc_debug_fieldop(int op, const uint64_t *d_a, const uint64_t *d_b, uint64_t *d_out, uint64_t n,
                     void *cuda_stream);
/* Integer-multiply roofline microbenchmark: runs `iters` dependent fp61 multiplies in each of `ilp`
 * independent chains per thread on grid x block threads; d_out receives one word per thread. */
int vc_bench_modmul(uint32_t grid, uint32_t block, uint32_t iters, uint32_t ilp, uint64_t *d_out, void *cuda_stream);

/* Per-kernel-kind device timing (bench.py's roofline): when enabled, every launch is bracketed by CUDA events on
 * its stream; vc_profile_read synchronises the device, sums launches and milliseconds per kind into two arrays of
 * VC_K_COUNT entries, and clears the records.  Enabling costs host time per launch: never on during a timed step. */
enum { VC_K_EVAL = 0, VC_K_SETUP = 1, VC_K_ROUND = 2, VC_K_UPDATE = 3, VC_K_LINE = 4, VC_K_FUSED_NARROW = 5,
       VC_K_FUSED_WIDE = 6, VC_K_MISC = 7, VC_K_FUSED_THIN = 8, VC_K_CLUSTER = 9, VC_K_COUNT = 10 };
int vc_profile_enable(int on);
int vc_profile_read(uint64_t *launches, double *ms);

#ifdef __cplusplus
}
#endif
#endif /* VC_H */
