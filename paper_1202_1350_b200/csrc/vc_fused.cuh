// vc_fused.cuh — the on-chip ("fused") schedule: ONE persistent cooperative kernel walks a range of layers;
// the per-gate state (weight P, fixed operand, packed record) of a layer stays in shared memory across all of
// its rounds, the three round values are all-reduced through one 64-byte L2 line per round, and every CTA draws
// the challenge itself, so a round costs one grid-wide rendezvous and no kernel launch.
//
// Same method as the streaming schedule (every gate contributes independently to every
// message); what changes is where the data lives and how the chain of dependent rounds
// is synchronised (SURVEY.md §7 "Round latency, not bandwidth, is the first wall").
//
// Layers with at most 2^10 gates and a table of at most 2^12 words are proved by CTA 0 alone out of shared
// memory (block barriers only) while the other CTAs wait at the next grid rendezvous.
#pragma once
#include "vc_kernels.cuh"
#include "vc_line.cuh"
#include "vc_round.cuh"

namespace vc {

constexpr int FT = 1024;                 // threads per CTA
constexpr int F_CHUNK_LOG = 10;          // a chunk = 1024 consecutive gates = one gate per thread
constexpr int F_MAXK = 8;                // chunks per CTA that fit in shared memory
constexpr int F_SMALL_N_LOG = 10;        // single-CTA path: gates <= 2^10 ...
constexpr int F_SMALL_T_LOG = 12;        // ... and table <= 2^12 words
constexpr int F_SLOT_WORDS = 128;        // one rendezvous slot: up to 64 values x (lo,hi)
constexpr int F_RING = 4;
constexpr uint64_t F_CNT_ONE = 1ull << 48;
constexpr uint64_t F_VAL_MASK = F_CNT_ONE - 1;

struct LayerDesc {
    const uint8_t *type;
    const uint32_t *in1, *in2;
    const uint64_t *V;       // values of this layer (entry d: the input)
    uint32_t log_n, pad;
};

struct FusedArgs {
    const LayerDesc *L;      // d+1 descriptors
    uint32_t d, begin, end;  // prove layers [begin, end)
    uint64_t seed;
    DevState *st;
    uint64_t *tr;            // transcript position of layer `begin`
    uint64_t *P, *T0, *T1;   // global scratch (streaming-mode weights; fold tables)
    unsigned long long *slots;  // F_RING * F_SLOT_WORDS words, all zero between launches
    uint64_t *stamps;        // d+1 words: %globaltimer (ns) when CTA 0 starts layer i, [d] = end of the proof
};

struct FusedCtx {            // block-shared bookkeeping, replicated in every CTA
    uint64_t z[MAX_VARS], r1[MAX_VARS], r2[MAX_VARS], q[MAX_VARS + 1];
    uint64_t acc[MAX_VARS];
    uint64_t red[3 * 32];
    uint64_t G[4];
    uint64_t seed, ctr, claim, v1, v2;
    uint32_t epoch, pad;
};

constexpr size_t F_STATE_BYTES = (size_t)F_MAXK * FT * (8 + 8 + 4 + 4);
constexpr size_t F_SMEM_BYTES = sizeof(FusedCtx) + F_STATE_BYTES;

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

// ---- grid rendezvous + all-reduce of K <= 64 canonical words (one per thread k < K, value in cx.acc[k]).
// Every CTA adds (value & 2^32-1 | 1<<48) and (value >> 32 | 1<<48) into the slot of this epoch; a word is
// complete when its count field equals the number of CTAs.  Totals land in cx.acc[k] of every CTA.
// All global writes made by this CTA before the call are visible to every CTA after it (fence + acquire).
__device__ __forceinline__ void grid_allreduce(FusedCtx &cx, const FusedArgs &a, uint32_t K) {
    const uint32_t tid = threadIdx.x;
    __syncthreads();
    unsigned long long *slot = a.slots + (size_t)(cx.epoch % F_RING) * F_SLOT_WORDS;
    if (blockIdx.x == 0 && tid >= 128 && tid < 128 + F_SLOT_WORDS)   // recycle the slot of epoch+2
        (a.slots + (size_t)((cx.epoch + 2) % F_RING) * F_SLOT_WORDS)[tid - 128] = 0ull;
    const uint32_t W = K == 0 ? 1 : 2 * K;
    uint64_t got = 0;
    if (tid < W) {
        const uint64_t v = K == 0 ? 0 : cx.acc[tid >> 1];
        const uint64_t part = (tid & 1) ? (v >> 32) : (v & 0xffffffffull);
        __threadfence();
        red_add(slot + tid, part | F_CNT_ONE);
        const uint64_t want = (uint64_t)gridDim.x;
        unsigned long long w;
        while (((w = ld_acquire(slot + tid)) >> 48) != want) { }
        got = w & F_VAL_MASK;
    }
    // combine lo + hi*2^32 (lo < 2^40, hi < 2^37)
    const uint64_t hi = __shfl_down_sync(0xffffffffu, got, 1);
    __syncthreads();
    if (tid < W && !(tid & 1) && K)
        cx.acc[tid >> 1] = fp61::add(fp61::reduce62(got), fp61::mul(hi, 1ull << 32));
    if (tid == 0) cx.epoch += 1;
    __syncthreads();
}

// block-level sum of 3 words per thread -> cx.acc[0..2] on every thread's view (after the trailing barrier)
__device__ __forceinline__ void block_reduce3(FusedCtx &cx, uint64_t (&v)[3]) {
    block_sum<3>(v, cx.red);
    if (threadIdx.x == 0) { cx.acc[0] = v[0]; cx.acc[1] = v[1]; cx.acc[2] = v[2]; }
    __syncthreads();
}

// Elo[u] = eq(u, z[0..c)) for u < 2^c, by doubling (1 multiply per new entry); c <= 10.  Trailing barrier.
__device__ __forceinline__ void build_eq_low(uint64_t *E, const uint64_t *z, uint32_t c) {
    if (threadIdx.x == 0) E[0] = 1;
    __syncthreads();
    for (uint32_t k = 0; k < c; k++) {
        const uint32_t half = 1u << k;
        if (threadIdx.x < half) {
            const uint64_t e = E[threadIdx.x], h = fp61::mul(e, z[k]);
            E[threadIdx.x + half] = h;
            E[threadIdx.x] = fp61::sub(e, h);
        }
        __syncthreads();
    }
}

// ---- a7, fused: cx.acc[t-2] <- sum over this CTA's share of V_{i+1} of eq(u, l(t)) V[u],  t = 2..s.
// One pass over the CTA's virtual blocks (2^(3+tb) words each, tb = min(s-3,10) thread bits): a thread folds its 8
// words with l(t)_{0..2}, weights by eq(lane bits), the warp sum is weighted by eq(warp bits, block bits).
// scratch: pts[m*s] | Wl[m*32] | Ww[m*32] | red[m*32]   (m = s-1 <= 63)
__device__ __forceinline__ void line_partials(const uint64_t *__restrict__ Vb, uint32_t s, FusedCtx &cx, uint64_t *scratch,
                                              uint32_t vb0, uint32_t vbstride) {
    const uint32_t m = s - 1, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    uint64_t *pts = scratch, *Wl = pts + (size_t)m * s, *Ww = Wl + (size_t)m * 32, *red = Ww + (size_t)m * 32;
    const uint32_t nt = s < 3 ? s : 3;
    const uint32_t tb = (s - nt) < 10 ? (s - nt) : 10;
    const uint32_t lb = tb < 5 ? tb : 5, wb = tb - lb;
    const uint32_t nvb = 1u << (s - nt - tb);
    if (tid < m) cx.acc[tid] = 0;
    for (uint32_t i = tid; i < m * s; i += FT) {
        const uint32_t t = i / s + 2, k = i % s;
        pts[i] = fp61::add(cx.r1[k], fp61::mul(t, fp61::sub(cx.r2[k], cx.r1[k])));
    }
    __syncthreads();
    // lane tables do not depend on the block: Wl[t][l] = eq(l, pts[t][nt..nt+lb))
    for (uint32_t i = tid; i < m * 32; i += FT) {
        const uint32_t t = i >> 5, l = i & 31;
        uint64_t e = 1;
        for (uint32_t k = 0; k < lb; k++) e = fp61::mul(e, fp61::chi((l >> k) & 1u, pts[t * s + nt + k]));
        Wl[i] = (l < (1u << lb)) ? e : 0;
    }
    const bool active = tid < (1u << tb);
    for (uint32_t vb = vb0; vb < nvb; vb += vbstride) {
        __syncthreads();
        for (uint32_t i = tid; i < m * 32; i += FT) {   // Ww[t][w] = eq(w, warp bits) * eq(vb, block bits)
            const uint32_t t = i >> 5, w = i & 31;
            uint64_t e = 1;
            for (uint32_t k = 0; k < wb; k++) e = fp61::mul(e, fp61::chi((w >> k) & 1u, pts[t * s + nt + lb + k]));
            for (uint32_t k = nt + tb; k < s; k++) e = fp61::mul(e, fp61::chi((vb >> (k - nt - tb)) & 1u, pts[t * s + k]));
            Ww[i] = e;
        }
        uint64_t v[8];
        const size_t base = (((size_t)vb << tb) + tid) << nt;
#pragma unroll
        for (int e = 0; e < 8; e++) v[e] = (active && e < (1 << nt)) ? Vb[base + e] : 0;
        __syncthreads();
        for (uint32_t t = 0; t < m; t++) {
            uint64_t f[8];
#pragma unroll
            for (int e = 0; e < 8; e++) f[e] = v[e];
#pragma unroll
            for (int k = 0; k < 3; k++) {
                if (k < (int)nt) {
                    const uint64_t x = pts[t * s + k];
#pragma unroll
                    for (int e = 0; e < (8 >> (k + 1)); e++) f[e] = fold2(f[2 * e], f[2 * e + 1], x);
                }
            }
            uint64_t val = active ? fp61::mul(f[0], Wl[t * 32 + lane]) : 0;
            val = warp_sum(val);
            if (lane == 0) red[t * 32 + warp] = fp61::mul(val, Ww[t * 32 + warp]);
        }
        __syncthreads();
        if (tid < m) {
            uint64_t acc = cx.acc[tid];
            const uint32_t nw = active ? ((1u << tb) + 31) >> 5 : 0;
            for (uint32_t w = 0; w < (((1u << tb) + 31) >> 5); w++) acc = fp61::add(acc, red[tid * 32 + w]);
            (void)nw;
            cx.acc[tid] = acc;
        }
    }
    __syncthreads();
}

// after the totals q[2..s] sit in cx.acc[0..m): write q, draw tau, z <- l(tau), claim <- q(tau).  All CTAs run it
// (identical results); only `writer` stores the transcript.
__device__ __forceinline__ void line_finish(uint32_t s, FusedCtx &cx, const DevState *st, uint64_t *tr_q, bool writer) {
    const uint32_t tid = threadIdx.x;
    if (tid <= s) cx.q[tid] = tid == 0 ? cx.v1 : (tid == 1 ? cx.v2 : cx.acc[tid - 2]);
    __syncthreads();
    const uint64_t tau = fp61::draw(cx.seed, cx.ctr);
    if (writer && tid <= s) tr_q[tid] = cx.q[tid];
    uint64_t term = 0;
    if (tid <= s) {
        uint64_t num = 1;
        for (uint32_t mm = 0; mm <= s; mm++)
            if (mm != tid) num = fp61::mul(num, fp61::sub(tau, mm));
        const uint64_t dinv = fp61::mul(st->invfact[tid], st->invfact[s - tid]);
        term = fp61::mul(cx.q[tid], fp61::mul(num, dinv));
        if ((s - tid) & 1u) term = fp61::neg(term);
    }
    uint64_t tv[1] = {term};
    block_sum<1>(tv, cx.red);
    if (tid < s) cx.z[tid] = fold2(cx.r1[tid], cx.r2[tid], tau);
    if (tid == 0) { cx.claim = tv[0]; cx.ctr += 1; }
    __syncthreads();
}

}  // namespace vc
