// vc_fused.cuh — the on-chip ("fused") schedule: ONE persistent cooperative kernel walks all layers of the proof.
//
// Same method as the streaming schedule (every gate contributes independently to every message,
// contributions are reduced in F_p).  What changes is where the data lives and how the chain
// of strictly dependent rounds is synchronised (SURVEY.md §7 "Round latency, not bandwidth, is the first wall"):
//   * per-gate state (W, c, idx) stays in shared memory across all 2s rounds of a layer (the paper's "no-copying
//     approach", pushed one level further up the memory hierarchy);
//   * every gate's contribution is W * (x + c): for MULT the fixed operand is folded into the weight once per phase
//     (W = P * V[in2]), for ADD/SUB/RELAY it is the additive constant c, so the hot loop has no per-type branch and
//     costs 3 wide multiplies per gate-round;
//   * fold tables live in shared memory: each CTA folds the slice its gates read (levels < K) and, from level K on,
//     the whole (<= 2^10-entry) table, redundantly; level K-1 is published through L2 once per phase;
//   * a round ends in one grid rendezvous on a count word in L2 (atom.add + polling by one lane per CTA); warp 15 of
//     every CTA (the "reducer") sums the CTA's committed contributions mod p and adds them to the round's six data
//     words with red.add — while the next round is already running on the thin path, in the shadow of the rendezvous on
//     the wide path (where all sixteen warps own gates); no kernel launch, no host round-trip.
// A challenge is only ever used AFTER every contribution to the message it answers has been committed (causality of
// the interactive protocol), although the seeded generator would allow drawing it earlier; what is
// pipelined is the summation of the committed contributions into the three transcript words.
#pragma once
#include "vc_kernels.cuh"

namespace vc {

constexpr int FT = 512;                  // threads per CTA (128 registers each)
constexpr int F_TLOG = 10;               // the fully shared part of a fold table has 2^min(s, F_TLOG) entries
constexpr int F_EQLOG = 10;              // eq tables are built in halves of at most 2^10 entries
constexpr int F_SMALL_N_LOG = 8;         // single-CTA path: gates <= 2^8 (one per worker thread) ...
constexpr int F_SMALL_T_LOG = 12;        // ... and table <= 2^12 words
constexpr int F_SLOT_WORDS = 128;        // one rendezvous slot: up to 64 values x (lo,hi)
constexpr int F_RING = 8;                // slots are recycled two epochs ahead and converted up to two epochs late
constexpr uint64_t F_CNT_ONE = 1ull << 48;
constexpr uint64_t F_VAL_MASK = F_CNT_ONE - 1;
constexpr uint32_t F_IDX_MASK = 0x3fffffffu;   // indices are < 2^30; bit 31 of a packed index = "x ignored" (RELAY, phase 2)
constexpr int F_MODE_SLICE = 0, F_MODE_GLOBAL = 1;

struct CtaPlan {                         // per (wide layer, CTA), computed at load from the host copy of the records
    uint32_t g0, g1;                     // gates [g0, g1) of the layer
    uint32_t blo[2], nb[2];              // per phase: first level-K block its gates read, and how many
    uint32_t own_lo[2], own_n[2];        // per phase (LayerPlan::pub_slice): the entries of level K-1 this CTA publishes from its own slice
};

struct LayerPlan {
    const uint8_t *type;
    const uint32_t *in1, *in2;
    const uint64_t *V;                   // values of this layer (entry d: the input)
    const CtaPlan *cta;                  // gridDim entries (wide layers), else null
    uint32_t log_n;
    uint32_t kind;                       // 0: single CTA, 1: grid-wide
    uint32_t thin;                       // != 0: at most one gate per worker thread: vc_fused_thin.cuh; the value = lanes per gate (1 or 4)
    uint32_t resident;                   // 1: gate state in shared memory, 0: in global scratch
    uint32_t has_relay;                  // 1: the layer has RELAY gates (their x is ignored in phase 2)
    uint32_t wiring, type0;              // implicit wiring (W_TREE / W_SELF with the single gate type type0, W_FIELDS with `rule`) or W_GENERIC
    WireRule rule;
    uint32_t cap;                        // state capacity in gates (multiple of FT)
    uint32_t mode[2];                    // per phase: F_MODE_SLICE / F_MODE_GLOBAL
    uint32_t K[2];                       // per phase: first fully shared level
    uint32_t pub_slice[2];               // per phase: 1 = the CTAs' slices cover level K-1 of the whole table, so each CTA publishes the entries
                                         // it owns straight from its slice (no pass over V_{i+1} with an eq table)
    uint32_t xw, yw;                     // words of the two fold buffers
    uint32_t off_tab, off_scr, off_commit;   // byte offsets in dynamic shared memory (after the state)
};

// Implicit wiring (§5.2: for regular circuits the in-neighbours of gate g are
// computed from g instead of being read).  Recognised at load: in1 = 2g, in2 = 2g+1 (the add trees), in1 = in2 = g (the
// squaring layers), and everything the bit-field rule of vc_state.cuh covers (chain lanes, matrix product, sliding
// window); everything else reads its records.
constexpr uint32_t W_GENERIC = 0, W_TREE = 1, W_SELF = 2, W_FIELDS = 3;
struct Wires {
    const uint8_t *type;
    const uint32_t *in1, *in2;
    const WireRule *rule;
    uint32_t mode, t0;
    __device__ __forceinline__ explicit Wires(const LayerPlan &L) : type(L.type), in1(L.in1), in2(L.in2), rule(&L.rule), mode(L.wiring), t0(L.type0) {}
    // with the rule read from a copy (shared memory) instead of the plan in global memory
    __device__ __forceinline__ Wires(const LayerPlan &L, const WireRule *r) : type(L.type), in1(L.in1), in2(L.in2), rule(r), mode(L.wiring), t0(L.type0) {}
    __device__ __forceinline__ uint32_t field_index(uint32_t g, int which) const {
        uint32_t v = rule->c[which];
#pragma unroll
        for (uint32_t k = 0; k < 3; k++) {
            const uint4 f = *reinterpret_cast<const uint4 *>(&rule->f[which][k]);     // p0, m, q0
            v += ((g >> f.x) & f.y) << f.z;
        }
        return v & rule->mask[which];
    }
    __device__ __forceinline__ uint32_t field_type(uint32_t g) const { return rule->t[(g >> rule->tbit) & rule->tm]; }
    __device__ __forceinline__ void get(uint32_t g, uint32_t &i1, uint32_t &i2, uint32_t &t) const {
        if (mode == W_TREE) { i1 = 2 * g; i2 = 2 * g + 1; t = t0; }
        else if (mode == W_SELF) { i1 = g; i2 = g; t = t0; }
        else if (mode == W_FIELDS) { i1 = field_index(g, 0); i2 = field_index(g, 1); t = field_type(g); }
        else { i1 = __ldg(in1 + g); i2 = __ldg(in2 + g); t = __ldg(type + g); }
    }
    // one field at a time (the non-resident gate loop needs in1 alone in phase 1, in2 and the type in phase 2)
    __device__ __forceinline__ uint32_t in1_of(uint32_t g) const { return mode == W_TREE ? 2 * g : (mode == W_SELF ? g : (mode == W_FIELDS ? field_index(g, 0) : __ldg(in1 + g))); }
    __device__ __forceinline__ uint32_t in2_of(uint32_t g) const { return mode == W_TREE ? 2 * g + 1 : (mode == W_SELF ? g : (mode == W_FIELDS ? field_index(g, 1) : __ldg(in2 + g))); }
    __device__ __forceinline__ uint32_t type_of(uint32_t g) const { return mode == W_GENERIC ? __ldg(type + g) : (mode == W_FIELDS ? field_type(g) : t0); }
};

struct FusedArgs {
    const LayerPlan *L;      // d+1 descriptors
    uint32_t d, begin, end;  // prove layers [begin, end)
    uint64_t seed;
    DevState *st;
    uint64_t *tr;            // transcript position of layer `begin`
    uint64_t *P, *C;         // global scratch: non-resident gate state (W, c)
    uint64_t *T0, *T1;       // global fold tables (F_MODE_GLOBAL)
    uint64_t *Tg;            // published level K-1 (F_MODE_SLICE), 2^(F_TLOG+1) words
    unsigned long long *slots;  // F_RING * F_SLOT_WORDS words, all zero between launches
    uint64_t *stamps;        // d+1 words: %globaltimer (ns) when CTA 0 starts layer i, [d] = end of the proof
};

struct FusedCtx {            // block-shared bookkeeping, replicated in every CTA
    uint64_t z[MAX_VARS], r1[MAX_VARS], r2[MAX_VARS], q[MAX_VARS + 1];
    uint64_t acc[MAX_VARS];
    uint64_t red[32 * 4];    // per-warp partials of a round
    uint64_t G[4];
    uint64_t seed, ctr, claim, v1, v2;
    uint32_t epoch, pad;
    WireRule wrule;          // the current layer's bit-field wiring rule (copied from its plan when the layer starts)
    uint32_t pad2;
};

// fixed part of the dynamic shared memory: FusedCtx, then 1/k! for k <= MAX_VARS, then Pascal's triangle C(n,k),
// n,k < 32 (u32); the rest starts 16-byte aligned
constexpr size_t F_INVFACT_OFF = sizeof(FusedCtx);
constexpr size_t F_PASCAL_OFF = (F_INVFACT_OFF + (MAX_VARS + 1) * 8 + 15) & ~(size_t)15;
constexpr size_t F_FIXED_BYTES = F_PASCAL_OFF + 32 * 32 * 4;

// Optional fine-grained trace (compile with -DVC_TRACE): CTA 0 / thread 0 appends (code << 48 | SM clock) after the
// d+1 layer stamps; read back with vc_debug_layer_stamps' buffer via vc_debug_trace.  Off in the product build.
constexpr uint32_t F_TRACE_WORDS = 1u << 16;
#ifdef VC_TRACE
#define VC_TR(code)                                                                                          \
    do {                                                                                                     \
        if (blockIdx.x == 0 && threadIdx.x == 0 && cx.pad < F_TRACE_WORDS) {                                 \
            a.stamps[a.d + 1 + cx.pad] = ((uint64_t)(code) << 48) | ((uint64_t)clock64() & 0xffffffffffffull); \
            cx.pad++;                                                                                        \
        }                                                                                                    \
    } while (0)
static __device__ uint64_t *g_tr_stamps;
static __device__ uint32_t g_tr_d;
#define VC_TRL(code)                                                                                         \
    do {                                                                                                     \
        if (blockIdx.x == 0 && threadIdx.x == 0 && cx.pad < F_TRACE_WORDS) {                                 \
            g_tr_stamps[g_tr_d + 1 + cx.pad] = ((uint64_t)(code) << 48) | ((uint64_t)clock64() & 0xffffffffffffull); \
            cx.pad++;                                                                                        \
        }                                                                                                    \
    } while (0)
#else
#define VC_TR(code) do { } while (0)
#define VC_TRL(code) do { } while (0)
#endif

__device__ __forceinline__ uint64_t fold2(uint64_t a, uint64_t b, uint64_t r) {
    return fp61::add(a, fp61::mul(r, fp61::sub(b, a)));
}
__device__ __forceinline__ unsigned long long ld_acquire(const unsigned long long *p) {
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ uint64_t globaltimer_ns() {
    uint64_t t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
__device__ __forceinline__ void red_add(unsigned long long *p, unsigned long long v) {
    asm volatile("red.relaxed.gpu.global.add.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
// barrier among the first nthr threads of the CTA (nthr a multiple of 32); id 1 (id 0 is __syncthreads)
__device__ __forceinline__ void bar_n(uint32_t nthr) { asm volatile("bar.sync 1, %0;" ::"r"(nthr) : "memory"); }

// Sum over the full warp of canonical words; every lane gets the canonical total.  Three integer warp reductions
// (REDUX) on 27/27/7-bit pieces instead of five shuffle+add levels.
__device__ __forceinline__ uint64_t warp_sum61(uint64_t v) {
    uint32_t p0 = (uint32_t)v & 0x7ffffffu, p1 = (uint32_t)(v >> 27) & 0x7ffffffu, p2 = (uint32_t)(v >> 54);
    p0 = __reduce_add_sync(0xffffffffu, p0);
    p1 = __reduce_add_sync(0xffffffffu, p1);
    p2 = __reduce_add_sync(0xffffffffu, p2);          // < 2^12
    const uint64_t x = (uint64_t)p0 + ((uint64_t)p1 << 27) + ((uint64_t)(p2 & 127u) << 54) + (p2 >> 7);
    return fp61::reduce62(x);                          // x < 2^32 + 2^59 + 2^61 + 32
}

// eq(u, x[k0..k1)) for one index u by direct product, two interleaved chains (no table, no barrier)
__device__ __noinline__ uint64_t eq_direct(uint32_t u, const uint64_t *x, uint32_t k0, uint32_t k1) {
    uint64_t e0 = 1, e1 = 1;
    uint32_t k = k0;
    for (; k + 1 < k1; k += 2) {
        e0 = fp61::mul(e0, fp61::chi((u >> (k - k0)) & 1u, x[k]));
        e1 = fp61::mul(e1, fp61::chi((u >> (k + 1 - k0)) & 1u, x[k + 1]));
    }
    if (k < k1) e0 = fp61::mul(e0, fp61::chi((u >> (k - k0)) & 1u, x[k]));
    return fp61::mul(e0, e1);
}

// Two-level eq table over variables x[0..nv): lo[u] = eq(u, x[0..cl)), hi[w] = eq(w, x[cl..ch)), cl = min(nv,10),
// ch = min(nv,20); variables >= 20 are multiplied in per index by eq_of().  Threads [t0, t0+nthr) cooperate; the
// caller provides the barrier afterwards.
struct EqTab {
    const uint64_t *lo, *hi, *x;
    uint32_t nv;
    __device__ __forceinline__ uint64_t eq_of(uint32_t u) const {
        uint64_t e = lo[u & ((1u << F_EQLOG) - 1)];
        if (nv > F_EQLOG) e = fp61::mul(e, hi[(u >> F_EQLOG) & ((1u << F_EQLOG) - 1)]);
        if (nv > 2 * F_EQLOG) e = fp61::mul(e, eq_direct(u >> (2 * F_EQLOG), x, 2 * F_EQLOG, nv));
        return e;
    }
};
// eq table over nv <= 10 variables as the outer product of two tables of <= 5 variables each (built by direct
// product in tmp[0..64)): one multiply per entry instead of nv.  Contains one block barrier; caller syncs afterwards.
__device__ __noinline__ void build_eq10(uint64_t *out, uint64_t *tmp, const uint64_t *x, uint32_t k0, uint32_t nv,
                                           uint32_t t, uint32_t nthr) {
    const uint32_t na = nv < 5 ? nv : 5, nb = nv - na;
    if (t < 64) {
        const uint32_t which = t >> 5, u = t & 31;
        if (which == 0) { if (u < (1u << na)) tmp[u] = eq_direct(u, x, k0, k0 + na); }
        else if (u < (1u << nb)) tmp[32 + u] = eq_direct(u, x, k0 + na, k0 + nv);
    }
    __syncthreads();
    for (uint32_t u = t; u < (1u << nv); u += nthr) out[u] = fp61::mul(tmp[u & ((1u << na) - 1)], tmp[32 + (u >> na)]);
}
// caller provides the barrier afterwards; tmp: 128 words of scratch
__device__ __noinline__ EqTab build_eq_tab(uint64_t *lo, uint64_t *hi, uint64_t *tmp, const uint64_t *x, uint32_t nv,
                                              uint32_t t, uint32_t nthr) {
    const uint32_t cl = nv < F_EQLOG ? nv : F_EQLOG;
    const uint32_t ch = nv < 2 * F_EQLOG ? nv : 2 * F_EQLOG;
    // both halves share the barrier: the 5-variable tables of the high half are built in tmp[64..128)
    const uint32_t na = cl < 5 ? cl : 5, nb = cl - na, hv = ch - cl, ha = hv < 5 ? hv : 5, hb = hv - ha;
    if (t < 128) {
        const uint32_t which = t >> 5, u = t & 31;
        if (which == 0) { if (u < (1u << na)) tmp[u] = eq_direct(u, x, 0, na); }
        else if (which == 1) { if (u < (1u << nb)) tmp[32 + u] = eq_direct(u, x, na, cl); }
        else if (which == 2) { if (u < (1u << ha)) tmp[64 + u] = eq_direct(u, x, cl, cl + ha); }
        else if (u < (1u << hb)) tmp[96 + u] = eq_direct(u, x, cl + ha, ch);
    }
    __syncthreads();
    for (uint32_t u = t; u < (1u << cl); u += nthr) lo[u] = fp61::mul(tmp[u & ((1u << na) - 1)], tmp[32 + (u >> na)]);
    if (hv) for (uint32_t u = t; u < (1u << hv); u += nthr) hi[u] = fp61::mul(tmp[64 + (u & ((1u << ha) - 1))], tmp[96 + (u >> ha)]);
    EqTab e; e.lo = lo; e.hi = hi; e.x = x; e.nv = nv;
    return e;
}

// ---- grid rendezvous + all-reduce of K <= 64 canonical words held in cx.acc[0..K) (CTA totals).
// Every CTA adds (low 32 bits | 1<<48) and (high bits | 1<<48) into the slot of this epoch; a word is complete when
// its count field equals the number of CTAs.  Totals land in cx.acc[k] of every CTA.  With fence = true all global
// writes made by this CTA before the call are visible to every CTA after it.
__device__ __noinline__ void grid_allreduce(FusedCtx &cx, const FusedArgs &a, uint32_t K, bool fence) {
    const uint32_t tid = threadIdx.x;
    __syncthreads();
    const uint32_t ep = cx.epoch;
    unsigned long long *slot = a.slots + (size_t)(ep % F_RING) * F_SLOT_WORDS;
    if (blockIdx.x == 0 && tid >= 128 && tid < 128 + F_SLOT_WORDS) {  // recycle the slot of epoch+2
        (a.slots + (size_t)((ep + 2) % F_RING) * F_SLOT_WORDS)[tid - 128] = 0ull;
        __threadfence();                 // ordered before CTA 0's post of epoch+1 (barrier below), hence before any post to it
    }
    const uint32_t W = K == 0 ? 1 : 2 * K;
    uint64_t got = 0;
    if (tid < W) {
        const uint64_t v = K == 0 ? 0 : cx.acc[tid >> 1];
        const uint64_t part = (tid & 1) ? (v >> 32) : (v & 0xffffffffull);
        if (fence) __threadfence();
        red_add(slot + tid, part | F_CNT_ONE);
        const uint64_t want = (uint64_t)gridDim.x;
        unsigned long long w;
        while (((w = ld_acquire(slot + tid)) >> 48) != want) { }
        got = w & F_VAL_MASK;
    }
    const uint64_t hi = __shfl_down_sync(0xffffffffu, got, 1);
    __syncthreads();
    if (tid < W && !(tid & 1) && K)
        cx.acc[tid >> 1] = fp61::add(fp61::reduce62(got), fp61::mul(hi, 1ull << 32));
    if (tid == 0) cx.epoch += 1;
    __syncthreads();
}

__device__ __forceinline__ unsigned long long atom_add(unsigned long long *p, unsigned long long v) {
    unsigned long long r;
    asm volatile("atom.relaxed.gpu.global.add.u64 %0, [%1], %2;" : "=l"(r) : "l"(p), "l"(v) : "memory");
    return r;
}
__device__ __forceinline__ unsigned long long ld_relaxed(const unsigned long long *p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}

// ---- warp-specialised rounds: vc_fused_thin.cuh has warps 0..14 work and warp 15 reduce beside them; vc_fused_wide.cuh
// gives gates to all sixteen warps and splits the round's upkeep (rendezvous, reduction, transcript) over warps 0, 15, 14.
constexpr uint32_t F_WORKERS = FT - 32;          // threads of warps 0..14
__device__ __forceinline__ void bar_workers() { asm volatile("bar.sync 2, %0;" ::"r"(F_WORKERS) : "memory"); }
// (hi:lo) += v if pred
__device__ __forceinline__ void add_c(uint64_t &lo, uint32_t &hi, uint64_t v, uint32_t pred) {
    asm("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %3, 0;\n\t@p add.cc.u64 %0, %0, %2;\n\t@p addc.u32 %1, %1, 0;\n\t}"
        : "+l"(lo), "+r"(hi) : "l"(v), "r"(pred));
}
// round slot: word 0 = count only (the rendezvous), words 1..6 = (low 32 | count), (high | count) of G0, G1, G2
__device__ __forceinline__ void round_slot_to_transcript(const unsigned long long *slot, uint64_t *tr, uint32_t lane) {
    uint64_t got = 0;
    if (lane >= 1 && lane < 7) {
        const uint64_t want = (uint64_t)gridDim.x;
        unsigned long long w;
        while (((w = ld_relaxed(slot + lane)) >> 48) != want) { }
        got = w & F_VAL_MASK;
    }
    const uint64_t hi = __shfl_down_sync(0xffffffffu, got, 1);
    if (lane >= 1 && lane < 7 && (lane & 1)) tr[(lane - 1) >> 1] = fp61::add(fp61::reduce62(got), fp61::mul(hi, 1ull << 32));
}
// warp 0, after the commit barrier: the rendezvous on the count word; the challenge is handed out afterwards.
// Memory-model note: the poll is ld.relaxed.gpu with no acquire fence behind it unless the round publishes data
// (fence == true), although the recycling of slot epoch+2 is ordered through this rendezvous: the last CTA zero-stores the
// slot, __threadfence()s, passes a CTA barrier, and only then its warp 0 arrives here with atom.relaxed; every other CTA
// adds into that slot only after it has SEEN the full count.  Formally (PTX memory model) the observers would need an
// acquire; on this hardware both the zero-store (made visible at L2 by the fence before the arrival) and the later red.add
// are performed at the one L2 slice that owns the line, and the add is control-dependent on the poll, so it cannot be
// performed before the count it waited for.  -DVC_RDV_ACQ puts a fence.acq_rel.gpu behind every poll (the formally
// conforming variant): bit-identical results, +93 us per config-2 proof (1.294 -> 1.387 ms, 278 grid rounds) on the box.
__device__ __forceinline__ void round_rendezvous(const FusedArgs &a, uint32_t ep, bool fence, uint64_t *rslot, uint64_t seed,
                                                 uint32_t ctr) {
    const uint64_t r = fp61::draw(seed, ctr);
    if ((threadIdx.x & 31) == 0) {
        unsigned long long *slot = a.slots + (size_t)(ep % F_RING) * F_SLOT_WORDS;
        if (fence) __threadfence();
        const uint64_t want = (uint64_t)gridDim.x;
        if ((atom_add(slot, F_CNT_ONE) >> 48) + 1 != want)
            while ((ld_relaxed(slot) >> 48) != want) { }
#ifdef VC_RDV_ACQ
        __threadfence();
#else
        if (fence) __threadfence();
#endif
        *rslot = r;
    }
}
// the reducer's bookkeeping in CTA 0: transcript positions of the last two rounds whose slots are not converted yet
struct RoundPend { uint64_t *tr1, *tr2; uint32_t s1, s2; };
// warp 15: the CTA totals t0..t2 (all lanes) go to the round's data words; CTA 0 converts the slot of two rounds ago
// into transcript words and recycles the slot of epoch+2
// the CTA totals t0..t2 (all lanes of the calling warp) are added to the round's six data words
__device__ __forceinline__ void reducer_post_data(const FusedArgs &a, uint32_t ep, uint64_t t0, uint64_t t1, uint64_t t2) {
    const uint32_t lane = threadIdx.x & 31;
    unsigned long long *slot = a.slots + (size_t)(ep % F_RING) * F_SLOT_WORDS;
    if (lane >= 1 && lane < 7) {
        const uint32_t k = (lane - 1) >> 1;
        const uint64_t v = k == 0 ? t0 : (k == 1 ? t1 : t2);
        red_add(slot + lane, (((lane - 1) & 1) ? (v >> 32) : (v & 0xffffffffull)) | F_CNT_ONE);
    }
}
// one warp per CTA: CTA 0 converts the slot of two rounds ago into transcript words, the last CTA recycles the slot of epoch+2
__device__ __forceinline__ void reducer_housekeeping(const FusedArgs &a, uint32_t ep, uint64_t *tr, RoundPend &pd) {
    const uint32_t lane = threadIdx.x & 31;
    if (blockIdx.x == 0) {
        if (pd.tr2) round_slot_to_transcript(a.slots + (size_t)pd.s2 * F_SLOT_WORDS, pd.tr2, lane);
        pd.tr2 = pd.tr1; pd.s2 = pd.s1; pd.tr1 = tr; pd.s1 = ep % F_RING;
    }
    if (blockIdx.x == gridDim.x - 1) {
        unsigned long long *z = a.slots + (size_t)((ep + 2) % F_RING) * F_SLOT_WORDS;
#pragma unroll
        for (int q = 0; q < F_SLOT_WORDS / 32; q++) z[q * 32 + lane] = 0ull;
        __threadfence();
    }
}
__device__ __forceinline__ void reducer_post(const FusedArgs &a, uint32_t ep, uint64_t t0, uint64_t t1, uint64_t t2, uint64_t *tr,
                                             RoundPend &pd) {     // the thin path's reducer warp does both jobs
    reducer_post_data(a, ep, t0, t1, t2);
    reducer_housekeeping(a, ep, tr, pd);
}
__device__ __forceinline__ void reducer_flush(const FusedArgs &a, RoundPend &pd) {
    const uint32_t lane = threadIdx.x & 31;
    if (blockIdx.x == 0) {
        if (pd.tr2) round_slot_to_transcript(a.slots + (size_t)pd.s2 * F_SLOT_WORDS, pd.tr2, lane);
        if (pd.tr1) round_slot_to_transcript(a.slots + (size_t)pd.s1 * F_SLOT_WORDS, pd.tr1, lane);
    }
    pd.tr1 = pd.tr2 = nullptr;
}

}  // namespace vc
