// vc_cluster.cuh — layers of at most 2^12 gates (CL_MAX_N) proved by ONE thread-block cluster (steps a2-a7).
//
// Same method as every other schedule (each gate contributes independently to each message, the
// contributions are reduced in F_p).  What this engine changes is the cost of the 2s strictly dependent
// rounds of a small layer ("several dozen messages": message j+1 needs challenge j) and of the
// per-layer work around them, which dominate the time of every layer below ~2^14 gates:
//   * a layer runs on A = 1, 2, 4, 8 or 16 CTAs of a 16-CTA cluster, one gate per thread in registers (W, c, idx, P);
//   * the end of a round is a COMMIT: every gate thread stores its two products to shared memory and the CTA's barrier
//     closes.  With A = 1 that barrier is the hand-off.  With A > 1 one lane per peer then arrives on the peer's
//     mbarrier through distributed shared memory (relaxed: the arrive carries no data); a thread uses challenge j only
//     after its own CTA's mbarrier has seen the commits of all A CTAs: every contribution to message j exists before
//     r_j is used.  No polling of global memory, no atomics;
//   * the summation of the committed products (step a5) is pipelined behind the hand-off: a service warp (no gates) sums
//     its CTA's commit buffer mod p and sends three words to CTA 0's inbox with st.async (the bytes are counted by an
//     mbarrier of their own); CTA 0's service warp adds the A shares of the previous round and writes the transcript;
//   * fold tables live in shared memory.  With regular wiring a CTA's gates read an aligned block of 2^m entries of
//     V_{i+1}: the CTA folds its own block for levels < m, the A blocks' last pairs are gathered into every CTA with
//     the commit of round m-1 (st.async), and from level m on every CTA folds the whole (<= 32-entry) table itself.
//     Irregular wiring: every CTA holds the whole table (m = s);
//   * the line restriction (a7) is STREAMED through phase 2 by two line warps (16, 17): the fold tree of V_{i+1} along
//     l(t) = r1 + t (r2 - r1) needs challenge r2_k for its level k only, so level k is folded as soon as round k of
//     phase 2 has been handed off (a per-thread cubic over variables 0..2, continued to t = 2..s by finite differences,
//     then one multiply per (node, t) and level).  When the last challenge arrives one fold is left and q[2..s] follow
//     within a few hundred cycles, instead of a separate pass over V_{i+1} after the rounds.  With A > 1 every CTA folds
//     its own block and the s-1 weighted block values are exchanged among the A CTAs with st.async;
//   * every active CTA finishes the layer itself (tau, z <- l(tau), claim <- q(tau)); CTAs that join a wider layer
//     receive (z, claim, ctr) from CTA 0.
#pragma once
#include "vc_fused.cuh"
#include "vc_fused_line.cuh"
#include "vc_fused_small.cuh"

namespace vc {

constexpr int CL_GW = 256;                  // gate threads per CTA (warps 0..7): one gate each
constexpr int CL_FW = 256;                  // fold threads (warps 8..15): the fold tables and the challenges
constexpr int CL_GT = CL_GW + CL_FW;
constexpr int CL_LT = 64;                   // line threads (warps 16, 17)
constexpr int CL_T = CL_GT + CL_LT + 64;    // + the transcript warp (18) and the service warp (19): 640 threads keep 96 registers each
constexpr int CL_C = 16;                    // CTAs per cluster
constexpr uint32_t CL_MAX_M = 13;           // a CTA's level-0 slice: at most 2^13 entries
constexpr uint32_t CL_MAX_S = 14;           // table below: at most 2^14 entries
constexpr uint32_t CL_MAX_N = 12;           // gates: at most 2^12 (16 CTAs x 256)
constexpr uint32_t CL_LINE_NONE = 0, CL_LINE_STREAM = 1, CL_LINE_DIRECT = 2, CL_LINE_PASS = 3;

struct ClLayer {                            // load-time plan of one layer (A = 0: not run by this engine)
    uint32_t A;                             // active CTAs (power of two)
    uint32_t gpc;                           // gates per active CTA
    uint32_t ngt, nft;                      // gate threads (tid < ngt) and fold threads (256 <= tid < 256 + nft) that take part, multiples of 32
    uint32_t m[2];                          // per phase: log2 entries of a CTA's level-0 slice (== s: the whole table)
    uint32_t blk[2][CL_C];                  // per phase and CTA: its slice is entries [blk << m, (blk + 1) << m)
    uint32_t lmode;                         // how q[2..s] are computed: CL_LINE_*
    uint32_t sb;                            // line restriction: a CTA's block of V_{i+1} has 2^sb words (sb = s - log2 A)
    uint32_t ltb, lthr;                     // CL_LINE_PASS: log2 threads per block of 8 words, threads taking part
    uint32_t off_line;                      // byte offset of the line buffers in dynamic shared memory
};

struct ClArgs {
    const LayerPlan *L;                     // d+1 descriptors (shared with k_fused)
    const ClLayer *cl;                      // d plans
    uint32_t d, begin, end;                 // prove layers [begin, end)
    uint32_t csize;                         // CTAs in the cluster (16, or 8 on a device that refuses 16)
    uint64_t seed;
    DevState *st;
    uint64_t *tr;                           // transcript position of layer `begin`
    uint64_t *stamps;                       // d+1 words: %globaltimer when CTA 0 starts layer i
};

constexpr uint32_t CL_MAX_LAYERS = 24;      // layers per launch (their plans are copied to shared memory; longer runs are split by the host)
struct ClPlanS { ClLayer C; LayerPlan Lp; const uint64_t *Vb; uint32_t s, pad; };   // one layer's plan, the table below it and its log size

struct ClShared {
    FusedCtx cx;
    uint64_t invfact[MAX_VARS + 1];
    uint64_t pad0;
    uint32_t pas[32 * 32];
    alignas(16) uint64_t mb_rd[2];          // round hand-off: 16 arrivals per phase (16/A from each active CTA); unused when A = 1
    uint64_t mb_end[2];                     // layer end (A > 1): own expect_tx + the bytes of the A CTAs' line shares
    uint64_t mb_dat[8];                     // CTA 0: the A x 32 bytes of inbox slot k have landed
    uint64_t mb_gat[2];                     // per phase: the 2A entries of the gather buffer have landed
    uint64_t mb_state;                      // (z, claim, ctr) from CTA 0 for a CTA that joins a wider layer
    volatile uint32_t rounds_done;          // rounds of the current layer handed off so far (read by the line and service warps)
    volatile uint32_t svc_done;             // rounds of the current layer whose commit buffer the service warp has summed
    volatile uint32_t tr_done;              // CTA 0: rounds of the current layer the transcript warp has written
    uint32_t pad1;
    alignas(16) uint64_t inbox[8][CL_C][4]; // CTA 0: per round (mod 8: the service warps of the other CTAs run up to five rounds ahead of CTA 0's) and CTA: G0, G1, G2, start-claim share
    alignas(16) uint64_t qin[2][CL_C][16];  // per layer parity and CTA: q[2..s] shares
    alignas(16) uint64_t gat[2][64];        // per phase: level m-1 of the fold table, all blocks
    alignas(16) uint64_t state_in[MAX_VARS + 2];   // z[0..64), claim, ctr
    uint64_t eqlo[128], eqhi[128];          // beta(z, g) = eqlo[g & 127] eqhi[g >> 7]
    uint64_t dk[32];                        // Lagrange denominators of the nodes 0..s: (-1)^(s-k) / (k! (s-k)!)
    uint64_t lpts[32];                      // line warps: l(t)_k of the level being folded, t = 2..s
    alignas(16) ClPlanS pl[CL_MAX_LAYERS];  // the plans of layers begin .. end-1
    alignas(16) ulonglong2 cbuf[4][CL_GW];  // committed products: a ring of four rounds (the service warp runs behind the gates)
    alignas(16) uint64_t chal[2][2];        // (r, 1 - r) of round jj in slot jj & 1: written by the dealer before the round's commit barrier,
                                            // read by everyone after the hand-off
#ifdef VC_TRACE
    uint32_t trc[768][8];                   // CTA 0 / thread 0: SM clock at marked points, one row per round or layer
    uint32_t trn;
    uint32_t trc2[64][4];
#endif
};

#ifdef VC_TRACE
#define CL_TRC(k) do { if (trace_thread) trow[k] = (uint32_t)clock64(); } while (0)
#define CL_TRC_ROW(tag) do { if (trace_thread && S.trn < 768) { trow[7] = (tag); for (int q_ = 0; q_ < 8; q_++) S.trc[S.trn][q_] = trow[q_]; S.trn++; } } while (0)
#else
#define CL_TRC(k) do { } while (0)
#define CL_TRC_ROW(tag) do { } while (0)
#endif

// ---- cluster / mbarrier primitives (PTX ISA: mapa, mbarrier, st.async; sm_90+)
__device__ __forceinline__ uint32_t cl_smem(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint32_t cl_mapa(uint32_t addr, uint32_t rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
    return r;
}
__device__ __forceinline__ uint32_t cl_rank() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ void cl_mbar_init(uint64_t *b, uint32_t cnt) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(cl_smem(b)), "r"(cnt) : "memory");
}
__device__ __forceinline__ void cl_mbar_expect(uint64_t *b, uint32_t bytes) {       // one arrival + bytes to come
    asm volatile("mbarrier.arrive.expect_tx.relaxed.cta.shared::cta.b64 _, [%0], %1;" ::"r"(cl_smem(b)), "r"(bytes) : "memory");
}
// The hand-off carries no data (what a peer learns is "this CTA has committed"; the data travels by st.async, whose bytes
// are counted by the mbarrier that guards them), so the arrive is relaxed: a release at cluster scope costs a
// MEMBAR.ALL.GPU per round.
__device__ __forceinline__ void cl_mbar_arrive_remote(uint32_t raddr, uint32_t cnt) {
    asm volatile("mbarrier.arrive.relaxed.cluster.shared::cluster.b64 _, [%0], %1;" ::"r"(raddr), "r"(cnt) : "memory");
}
__device__ __forceinline__ void cl_mbar_wait_relaxed(uint64_t *b, uint32_t parity) {
    asm volatile("{\n\t.reg .pred p;\n\tCLR: mbarrier.try_wait.parity.relaxed.cluster.shared::cta.b64 p, [%0], %1;\n\t@!p bra CLR;\n\t}"
                 ::"r"(cl_smem(b)), "r"(parity) : "memory");
}
__device__ __forceinline__ void cl_mbar_wait(uint64_t *b, uint32_t parity) {        // acquire: the counted bytes are visible afterwards
    asm volatile("{\n\t.reg .pred p;\n\tCLW: mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%0], %1;\n\t@!p bra CLW;\n\t}"
                 ::"r"(cl_smem(b)), "r"(parity) : "memory");
}
__device__ __forceinline__ void cl_st_async(uint32_t raddr, uint64_t v, uint32_t rmbar) {
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.b64 [%0], %1, [%2];" ::"r"(raddr), "l"(v), "r"(rmbar) : "memory");
}
__device__ __forceinline__ void cl_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ void cl_bar(uint32_t id, uint32_t nthr) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthr) : "memory"); }

// W (x + c) mod p up to a multiple of p, left unreduced: below 2^63 for W < 2^61, m < 2^62.6 and below 2^64 for m < 2^63
// (the committed words are summed in 96 bits by the service warp).
__device__ __forceinline__ uint64_t cl_mul_lazy(uint64_t W, uint64_t m) {
    const uint64_t lo = W * m, hi = fp61::mulhi(W, m);
    return (lo & fp61::P) + ((lo >> 61) | (hi << 3));
}
// service warp: the CTA's three sums of one message from its commit buffer (x | bit << 63, y').  Per lane three 96-bit
// sums (all x, x with bit 1, all y'); across the lanes REDUX on 27/27/19-bit pieces; lane k < 3 then assembles value k:
// lane 0: G0 = sum x - sum_{bit 1} x, lane 1: G1 = sum_{bit 1} x, lane 2: G2 = sum y'.  Returns this lane's value.
__device__ __noinline__ uint64_t cl_svc_sums(const ulonglong2 *cb, uint32_t gpc) {
    const uint32_t lane = threadIdx.x & 31;
    uint64_t Sl = 0, S1l = 0, Tl = 0; uint32_t Sh = 0, S1h = 0, Th = 0;
#pragma unroll 1
    for (uint32_t i = lane; i < gpc; i += 32) {
        const ulonglong2 q = cb[i];                          // (W (x_b + c) | bit << 63,  chi(bit, 2) W (x_2 + c)), both unreduced
        const uint32_t bit = (uint32_t)(q.x >> 63);
        const uint64_t v1 = q.x & ~(1ull << 63);
        add_c(Sl, Sh, v1, 1u); add_c(S1l, S1h, v1, bit); add_c(Tl, Th, q.y, 1u);
    }
    uint32_t pc[9];                                          // hi < 2^4 (at most 8 words per lane): top piece < 2^14, its sum < 2^19
    pc[0] = (uint32_t)Sl & 0x7ffffffu;  pc[1] = (uint32_t)(Sl >> 27) & 0x7ffffffu;  pc[2] = (uint32_t)(Sl >> 54) | (Sh << 10);
    pc[3] = (uint32_t)S1l & 0x7ffffffu; pc[4] = (uint32_t)(S1l >> 27) & 0x7ffffffu; pc[5] = (uint32_t)(S1l >> 54) | (S1h << 10);
    pc[6] = (uint32_t)Tl & 0x7ffffffu;  pc[7] = (uint32_t)(Tl >> 27) & 0x7ffffffu;  pc[8] = (uint32_t)(Tl >> 54) | (Th << 10);
#pragma unroll
    for (int k = 0; k < 9; k++) pc[k] = __reduce_add_sync(0xffffffffu, pc[k]);
    const uint32_t q = lane == 2 ? 2u : 1u;                  // lanes 0 and 1 assemble sum_{bit 1} x, lane 2 sum y'; lane 0 also sum x
    const uint32_t a0 = q == 2 ? pc[6] : pc[3], a1 = q == 2 ? pc[7] : pc[4], a2 = q == 2 ? pc[8] : pc[5];
    // 2^54 * a2 = 2^54 (a2 & 127) + 2^61 (a2 >> 7) = 2^54 (a2 & 127) + (a2 >> 7)  (mod p)
    uint64_t v = fp61::reduce62((uint64_t)a0 + ((uint64_t)a1 << 27) + ((uint64_t)(a2 & 127u) << 54) + (a2 >> 7));
    if (lane == 0) {
        const uint64_t x = fp61::reduce62((uint64_t)pc[0] + ((uint64_t)pc[1] << 27) + ((uint64_t)(pc[2] & 127u) << 54) + (pc[2] >> 7));
        v = fp61::sub(x, v);
    }
    return v;
}

struct ClPhases { uint32_t rd[2], gat[2], dat[8], end[2], state; };   // parity of the next phase to wait for, per mbarrier

// Round numbering.  R counts the rounds this CTA has taken part in since the launch (it indexes the commit ring and the
// counters rounds_done / svc_done); Q counts the rounds of layers run by more than one CTA (the same in every CTA: it
// indexes CTA 0's inbox ring and tr_done).
// ---- the service warp (a5, behind the gates): this CTA's sums of every message go to CTA 0's inbox (A > 1) or straight to
// the transcript (A = 1).  It follows the hand-offs through rounds_done and frees the commit buffers through svc_done;
// it runs through all layers of the launch on its own, a few messages behind the gates, and is on nobody's critical path.
__device__ __forceinline__ void cl_svc_role(const ClArgs &a, ClShared &S, uint32_t rank) {
    const uint32_t lane = threadIdx.x & 31;
    uint64_t *tr = a.tr;
    uint32_t R = 0, Q = 0;
    for (uint32_t layer = a.begin; layer < a.end; layer++) {
        const ClLayer &C = S.pl[layer - a.begin].C;
        const uint32_t s = S.pl[layer - a.begin].s, A = C.A, gpc = C.gpc, ngw = (gpc + 31) >> 5;
        if (rank < A) {
#pragma unroll 1
            for (uint32_t jj = 0; jj < 2 * s; jj++, R++) {
                while (S.rounds_done < R + 1) { }
                if (rank == 0 && A > 1) while (S.tr_done + 4 < Q + jj + 1) { }   // bounds how far the inbox writers run ahead
                uint64_t mine = cl_svc_sums(S.cbuf[R & 3], gpc);
                __syncwarp();
                if (lane == 0) S.svc_done = R + 1;
                if (layer == 0 && jj == 0) {                 // a2: the start claim's share rides with message 0
                    const uint64_t t3 = warp_sum61(lane < ngw ? S.cx.red[lane] : 0);
                    if (lane == 3) mine = t3;
                }
                if (A == 1) {                                // the CTA's sums are the message
                    if (lane < 3) tr[3 * jj + lane] = mine;
                    if (layer == 0 && jj == 0 && lane == 3) a.st->G[3] = mine;
                } else if (lane < 4) {
                    const uint32_t k = (Q + jj) & 7;
                    cl_st_async(cl_mapa(cl_smem(&S.inbox[k][rank][lane]), 0), mine, cl_mapa(cl_smem(&S.mb_dat[k]), 0));
                }
            }
        }
        if (A > 1) Q += 2 * s;
        tr += 7 * (size_t)s + 1;
    }
}
// ---- the transcript warp of CTA 0: message jj of a layer run by A > 1 CTAs = the sum of the A shares in its inbox slot
__device__ __forceinline__ void cl_tr_role(const ClArgs &a, ClShared &S) {
    const uint32_t lane = threadIdx.x & 31;
    uint64_t *tr = a.tr;
    uint32_t Q = 0, phase[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    for (uint32_t layer = a.begin; layer < a.end; layer++) {
        const uint32_t s = S.pl[layer - a.begin].s, A = S.pl[layer - a.begin].C.A;
        if (A > 1) {
#pragma unroll 1
            for (uint32_t jj = 0; jj < 2 * s; jj++, Q++) {
                const uint32_t k = Q & 7;
                if (lane == 0) cl_mbar_expect(&S.mb_dat[k], A * 32);
                cl_mbar_wait(&S.mb_dat[k], (phase[k] & 1u));
                phase[k] ^= 1u;
                const uint64_t g0 = warp_sum61(lane < A ? S.inbox[k][lane][0] : 0), g1 = warp_sum61(lane < A ? S.inbox[k][lane][1] : 0);
                const uint64_t g2 = warp_sum61(lane < A ? S.inbox[k][lane][2] : 0);
                if (lane < 3) tr[3 * jj + lane] = lane == 0 ? g0 : (lane == 1 ? g1 : g2);
                if (layer == 0 && jj == 0) {
                    const uint64_t g3 = warp_sum61(lane < A ? S.inbox[k][lane][3] : 0);
                    if (lane == 0) a.st->G[3] = g3;
                }
                __syncwarp();
                if (lane == 0) S.tr_done = Q + 1;
            }
        }
        tr += 7 * (size_t)s + 1;
    }
}

// The two-level eq table of r1 (S.eqlo over variables 0..6, S.eqhi over 7..s-1), grown by one variable per challenge:
// E[u + 2^k'] = E[u] r, E[u] -= E[u + 2^k'] for u < 2^k', k' = k mod 7 (one multiply per new entry).  Fold threads only;
// consecutive steps are separated by the round barriers.
__device__ __forceinline__ void cl_eq_step(ClShared &S, uint32_t k, uint64_t r, uint32_t ft, uint32_t nft) {
    uint64_t *E = k < 7 ? S.eqlo : S.eqhi;
    const uint32_t kk = k < 7 ? k : k - 7, half = 1u << kk;
    for (uint32_t u = ft; u < half; u += nft) {
        const uint64_t e = kk == 0 ? 1 : E[u], hi = fp61::mul(e, r);
        E[u + half] = hi;
        E[u] = fp61::sub(e, hi);
    }
}

// What a layer needs from global memory before its first round: the level-0 slices of both phases (cp.async into shared
// memory) and, per gate thread, its record and fixed operand (registers).  None of it depends on a challenge, so the
// loads of layer i+1 are issued while layer i finishes (tau, z, claim), or while a joining CTA waits for the state.
struct ClPre { uint32_t layer, i1, i2, t; uint64_t other; };
__device__ __forceinline__ void cl_cp16(void *dst_smem, const void *src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(cl_smem(dst_smem)), "l"(src) : "memory");
}
__device__ __forceinline__ void cl_fetch(const ClArgs &a, const ClShared &S, uint8_t *dyn, uint32_t layer, uint32_t rank, ClPre &pre) {
    const uint32_t tid = threadIdx.x;
    constexpr uint32_t NM = CL_T - 64;
    const ClPlanS &P = S.pl[layer - a.begin];
    const ClLayer &C = P.C;
    uint64_t *X = reinterpret_cast<uint64_t *>(dyn);
    const uint32_t mmax = C.m[0] > C.m[1] ? C.m[0] : C.m[1];
    uint64_t *Y = X + ((1u << mmax) < 64u ? 64u : (1u << mmax));
    uint64_t *X2 = Y + ((1u << (mmax - 1)) < 64u ? 64u : (1u << (mmax - 1)));
    {
        const uint64_t *src = P.Vb + ((size_t)C.blk[0][rank] << C.m[0]);
#pragma unroll 1
        for (uint32_t v = tid; v < (1u << (C.m[0] - 1)); v += NM) cl_cp16(X + 2 * v, src + 2 * v);
        src = P.Vb + ((size_t)C.blk[1][rank] << C.m[1]);
#pragma unroll 1
        for (uint32_t v = tid; v < (1u << (C.m[1] - 1)); v += NM) cl_cp16(X2 + 2 * v, src + 2 * v);
        asm volatile("cp.async.commit_group;" ::: "memory");
    }
    pre.layer = layer; pre.i1 = 0; pre.i2 = 0; pre.t = VC_RELAY; pre.other = 0;
    if (tid < C.gpc) {
        Wires(P.Lp).get(rank * C.gpc + tid, pre.i1, pre.i2, pre.t);
        pre.other = __ldg(P.Vb + pre.i2);
    }
}

// ---- the rounds of one layer in an active CTA, gate threads (tid < ngt) and fold threads (256 <= tid < 256 + nft).
// A gate thread's stream per round is: read the challenge, one multiply for the weight, wait for the level, read its
// pair, two products, commit.  The fold threads build the level meanwhile and one of them (the dealer) draws the next
// challenge while the gates form their products; the value is read by anyone only after the round's hand-off.
__device__ __forceinline__ void cl_rounds(const ClArgs &a, ClShared &S, uint8_t *dyn, uint32_t layer, uint32_t rank, uint32_t Rb,
                                          ClPhases &php, const ClPre &pre) {
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const LayerPlan &Lp = S.pl[layer - a.begin].Lp;
    const ClLayer &C = S.pl[layer - a.begin].C;
    const uint32_t si = Lp.log_n, s = S.pl[layer - a.begin].s, A = C.A, gpc = C.gpc, ngt = C.ngt, nft = C.nft, np = ngt + nft;
    const bool gate_thr = tid < CL_GW, has_ign = Lp.has_relay != 0;
    const uint32_t ft = tid - CL_GW;                         // fold thread number (fold threads only)
    const uint32_t pidx = gate_thr ? tid : ngt + ft;         // number among the np participants
    FusedCtx &cx = S.cx;
    const uint64_t seed = cx.seed;
    const uint32_t ctr0 = (uint32_t)cx.ctr;
    const uint32_t arr_cnt = CL_C / A;                       // every active CTA contributes 16/A of the 16 arrivals
    const bool live = gate_thr && tid < gpc;
    const uint32_t g = rank * gpc + (live ? tid : 0);
    uint64_t *X = reinterpret_cast<uint64_t *>(dyn);          // level 0 of phase 1, then the even levels of both phases
    const uint32_t mmax = C.m[0] > C.m[1] ? C.m[0] : C.m[1];
    uint64_t *Y = X + ((1u << mmax) < 64u ? 64u : (1u << mmax));          // the odd levels
    uint64_t *X2 = Y + ((1u << (mmax - 1)) < 64u ? 64u : (1u << (mmax - 1)));   // level 0 of phase 2, fetched while phase 1 runs
#ifdef VC_TRACE
    const bool trace_thread = rank == 0 && tid == 0;
    uint32_t trow[8] = {0, 0, 0, 0, 0, 0, 0, 0};
#endif

    // ---- a3 and the phase-1 state of this thread's gate (record, fixed operand and slices were fetched ahead: cl_fetch)
    const uint32_t i1 = pre.i1, i2 = pre.i2, t = pre.t;
    uint32_t idx = 0;
    uint64_t W = 0, cP = fp61::P, P = 0;
    const uint64_t other = pre.other;
    CL_TRC(0);
    if (si <= 6) {
        if (live) P = eq_direct(g, cx.z, 0, si);
    } else {
        const uint32_t nl = 7, nh = si - 7;
#pragma unroll 1
        for (uint32_t e = pidx; e < 128 + (1u << nh); e += np) {
            if (e < 128) S.eqlo[e] = eq_direct(e, cx.z, 0, nl);
            else S.eqhi[e - 128] = eq_direct(e - 128, cx.z, nl, si);
        }
        cl_bar(2, np);
        if (live) P = fp61::mul(S.eqlo[g & 127u], S.eqhi[g >> 7]);
    }
    CL_TRC(1);
    if (live) {
        uint64_t c; uint32_t ign;
        gate_state(1, t, P, other, W, c, ign);
        cP = c + fp61::P; idx = i1;
    }
    CL_TRC(2);
    if (layer == 0 && gate_thr) {                            // a2: this CTA's share of the start claim V~_0(z_0)
        const uint64_t part = warp_sum61(live ? fp61::mul(P, __ldg(Lp.V + g)) : 0);
        if (lane == 0) cx.red[warp] = part;
    }

    uint32_t jj = 0;                                         // round number within the layer, 0 .. 2s-1
    for (int ph = 0; ph < 2; ph++) {
        const uint32_t m = C.m[ph], blk = C.blk[ph][rank];
        const bool sliced = m < s;
        if (sliced && tid == 0) cl_mbar_expect(&S.mb_gat[ph], 2 * A * 8);
        if (ph == 1) {
            CL_TRC_ROW(1000u * layer + 901u);
            CL_TRC(0);
            // ---- phase switch: V~(r1) from the last level, P = beta(z,g) eq(in1[g], r1) through a two-level eq table of r1,
            // the phase-2 state, the new slice
            const uint64_t *t1 = s == 1 ? X : (((s - 1) & 1) ? Y : X);     // the last level of phase 1
            const uint64_t v1 = fold2(t1[0], t1[1], S.chal[(jj - 1) & 1][0]);
            if (tid == 0) cx.v1 = v1;
            if (!gate_thr) cl_eq_step(S, s - 1, S.chal[(jj - 1) & 1][0], ft, nft);   // the last variable of the eq table of r1
            CL_TRC(1);
            cl_bar(2, np);                                   // everyone has read the last level of phase 1; the eq table of r1 is complete
            CL_TRC(2);
            if (live) {
                const uint32_t nl = s < 7 ? s : 7;
                const uint64_t e1 = s > nl ? fp61::mul(S.eqlo[i1 & ((1u << nl) - 1)], S.eqhi[i1 >> nl]) : S.eqlo[i1];
                P = fp61::mul(P, e1);
                uint64_t c; uint32_t ign;
                gate_state(2, t, P, v1, W, c, ign);
                cP = c + fp61::P; idx = i2 | (ign << 31);
            }
        }
        CL_TRC(3);
        if (ph == 0) asm volatile("cp.async.wait_all;" ::: "memory");
        cl_bar(2, np);                                       // level 0 is in place
        CL_TRC(4);
        CL_TRC_ROW(1000u * layer + 900u + 2u * ph);
        CL_TRC(0);
#pragma unroll 1
        for (uint32_t j = 0; j < s; j++, jj++) {
            const uint32_t par = jj & 1;
            const uint64_t *L0 = ph ? X2 : X;
            const uint64_t *tab = j == 0 ? L0 : ((j & 1) ? Y : X);   // level j as this CTA holds it
            if (gate_thr) {
                if (j >= 1) {
                    // ---- a6 for the challenge of the previous round: this gate's weight
                    const ulonglong2 ch = *reinterpret_cast<const ulonglong2 *>(S.chal[(jj - 1) & 1]);
                    if (live) W = fp61::mul(W, ((idx >> (j - 1)) & 1u) ? ch.x : ch.y);
                    cl_bar(2, np);                           // level j is complete
                }
                CL_TRC(1);
                if (sliced && j == m - 1 && tid < 2 * A)     // this block's last pair goes to every CTA's gather buffer
                    cl_st_async(cl_mapa(cl_smem(&S.gat[ph][2 * blk + (tid & 1u)]), tid >> 1), tab[tid & 1u],
                                cl_mapa(cl_smem(&S.mb_gat[ph]), tid >> 1));
                // ---- a4: this thread's gate against level j
                if (live) {
                    const uint32_t bit = (idx >> j) & 1u, u = (idx & F_IDX_MASK) >> (j + 1);
                    const uint32_t pos = j < m ? 2 * u - (blk << (m - j)) : 2 * u;
                    const ulonglong2 p = *reinterpret_cast<const ulonglong2 *>(tab + pos);
                    uint64_t lo = p.x, hi = p.y;
                    if (has_ign && (idx >> 31)) { lo = 0; hi = 0; }
                    const uint64_t mb = (bit ? hi : lo) + cP, m2 = 2 * hi + cP - lo;
                    const uint64_t y = cl_mul_lazy(W, m2), yc = (y & fp61::P) + (y >> 61);      // < 2^61 + 8
                    ulonglong2 o;
                    o.x = cl_mul_lazy(W, mb) | ((uint64_t)bit << 63);
                    o.y = bit ? 2 * yc : 2 * fp61::P - yc;   // chi(bit, 2) W (x_2 + c), unreduced
                    while (S.svc_done + 4 < Rb + jj + 1) { }     // the ring slot is free (the service warp is rarely that far behind)
                    S.cbuf[(Rb + jj) & 3][tid] = o;
                }
            } else {
                if (j >= 1) {
                    // ---- a6: level j of the fold table from level j-1 and the challenge of the previous round
                    const uint64_t r_prev = S.chal[(jj - 1) & 1][0];
                    uint64_t *dst = (j & 1) ? Y : X;
                    const uint64_t *srcl = j == 1 ? L0 : (((j - 1) & 1) ? Y : X);
                    if (sliced && j == m) {                  // the first whole level comes from the gathered level m-1
                        cl_mbar_wait(&S.mb_gat[ph], php.gat[ph]);
                        srcl = S.gat[ph];
                    }
                    const uint32_t cnt = j < m ? 1u << (m - j) : 1u << (s - j);
#pragma unroll 1
                    for (uint32_t v = ft; v < cnt; v += nft) {
                        const ulonglong2 p = *reinterpret_cast<const ulonglong2 *>(srcl + 2 * (size_t)v);
                        dst[v] = fold2(p.x, p.y, r_prev);
                    }
                    cl_bar(2, np);
                    if (ph == 0) cl_eq_step(S, j - 1, r_prev, ft, nft);   // the eq table of r1 grows by variable j-1 while the gates form their products
                }
                if (ft == 0) {                               // the dealer: challenge jj, ready in shared memory before the commit barrier
                    const uint64_t r = fp61::draw(seed, ctr0 + jj);
                    ulonglong2 ch; ch.x = r; ch.y = fp61::sub(1, r);
                    *reinterpret_cast<ulonglong2 *>(S.chal[par]) = ch;
                }
            }
            CL_TRC(2);
            cl_bar(3, np);                                   // every contribution of this CTA to message jj is committed
            CL_TRC(3);
            if (A > 1) {
                if (warp == 0 && lane < A) cl_mbar_arrive_remote(cl_mapa(cl_smem(&S.mb_rd[par]), lane), arr_cnt);
                cl_mbar_wait_relaxed(&S.mb_rd[par], php.rd[par]);
                php.rd[par] ^= 1u;
            }
            if (tid == 0) S.rounds_done = Rb + jj + 1;       // the line and service warps may go on from here
            CL_TRC(4);
            CL_TRC_ROW(1000u * layer + jj);
            CL_TRC(0);
        }
        if (sliced) php.gat[ph] ^= 1u;
    }
    // ---- V~_{i+1}(r2) from the last level
    if (tid == 0) {
        const uint64_t *t1 = s == 1 ? X2 : (((s - 1) & 1) ? Y : X);    // the last level of phase 2
        cx.v2 = fold2(t1[0], t1[1], S.chal[(jj - 1) & 1][0]);
    }
}

// ---- a7, streamed: the line warps fold this CTA's block of V_{i+1} along l(t) = r1 + t (r2 - r1), one level per challenge
// of phase 2, and leave the block's weighted values q_c[t], t = 2..s, in cx.acc[t - 2].  (Reading c-5; the polynomial
// tree is that of vc_fused_line.cuh: a level-k node is a polynomial of degree k in t.)
__device__ __forceinline__ void cl_line_wait(const ClShared &S, uint32_t need) {
    while (S.rounds_done < need) { }
}
__device__ __forceinline__ void cl_line_stream(const ClArgs &a, ClShared &S, uint8_t *dyn, uint32_t layer, uint32_t rank, uint32_t Rb) {
    const uint32_t lt = threadIdx.x - CL_GT;                 // 0 .. CL_LT-1
    const ClLayer &C = S.pl[layer - a.begin].C;
    const uint32_t s = S.pl[layer - a.begin].s, sb = C.sb, m = s - 1;
    FusedCtx &cx = S.cx;
    const uint64_t seed = cx.seed;
    const uint32_t ctr0 = (uint32_t)cx.ctr;
    const uint64_t *__restrict__ Vblk = S.pl[layer - a.begin].Vb + ((size_t)rank << sb);
    uint64_t *LA = reinterpret_cast<uint64_t *>(dyn + C.off_line);
    if (C.lmode == CL_LINE_DIRECT) {
        // tiny blocks (fewer than 8 words): q_c[t] = sum_u eq(u, l(t)) V[u] by direct products, once every challenge is known
        cl_line_wait(S, Rb + 2 * s);
        if (lt < m) {
            const uint32_t t = lt + 2;
            uint64_t acc = 0;
            for (uint32_t u = 0; u < (1u << sb); u++) {
                const uint32_t e = (rank << sb) + u;
                uint64_t w = 1;
                for (uint32_t k = 0; k < s; k++) {
                    const uint64_t p = fp61::draw(seed, ctr0 + k), q = fp61::draw(seed, ctr0 + s + k);
                    const uint64_t x = fp61::add(p, fp61::mul(t, fp61::sub(q, p)));
                    w = fp61::mul(w, fp61::chi((e >> k) & 1u, x));
                }
                acc = fp61::add(acc, fp61::mul(w, __ldg(Vblk + u)));
            }
            cx.acc[lt] = acc;
        }
        return;
    }
    const uint32_t nE = 1u << (sb - 3);                      // nodes after the per-thread cubic stage
    uint64_t *LB = LA + (size_t)nE * m;
    // the first node's 8 words travel while phase 1 runs
    ulonglong2 w8[4];
    if (lt < nE) {
        const ulonglong2 *p2 = reinterpret_cast<const ulonglong2 *>(Vblk + ((size_t)lt << 3));
#pragma unroll
        for (int e = 0; e < 4; e++) w8[e] = __ldg(p2 + e);
    }
    cl_line_wait(S, Rb + s + 3);                             // r2_0..2 have been handed off
    uint64_t x[3][4];
#pragma unroll
    for (int k = 0; k < 3; k++) {
        const uint64_t p = fp61::draw(seed, ctr0 + k), q = fp61::draw(seed, ctr0 + s + k), d = fp61::sub(q, p);
        x[k][0] = p; x[k][1] = q; x[k][2] = fp61::add(q, d); x[k][3] = fp61::add(x[k][2], d);
    }
#pragma unroll 1
    for (uint32_t e0 = lt; e0 < nE; e0 += CL_LT) {
        if (e0 != lt) {
            const ulonglong2 *p2 = reinterpret_cast<const ulonglong2 *>(Vblk + ((size_t)e0 << 3));
#pragma unroll
            for (int e = 0; e < 4; e++) w8[e] = __ldg(p2 + e);
        }
        uint64_t v[8];
#pragma unroll
        for (int e = 0; e < 4; e++) { v[2 * e] = w8[e].x; v[2 * e + 1] = w8[e].y; }
        uint64_t f1[4][3];
#pragma unroll
        for (int e = 0; e < 4; e++) {
            const uint64_t d = fp61::sub(v[2 * e + 1], v[2 * e]);
            f1[e][0] = fp61::add(v[2 * e], fp61::mul(x[0][0], d));
            f1[e][1] = fp61::add(v[2 * e], fp61::mul(x[0][1], d));
            f1[e][2] = fp61::sub(fp61::dbl(f1[e][1]), f1[e][0]);
        }
        uint64_t f2[2][4];
#pragma unroll
        for (int e = 0; e < 2; e++) {
#pragma unroll
            for (int t = 0; t < 3; t++)
                f2[e][t] = fp61::add(f1[2 * e][t], fp61::mul(x[1][t], fp61::sub(f1[2 * e + 1][t], f1[2 * e][t])));
            const uint64_t d21 = fp61::sub(f2[e][2], f2[e][1]);
            f2[e][3] = fp61::add(fp61::add(fp61::dbl(d21), d21), f2[e][0]);
        }
        uint64_t f[4];
#pragma unroll
        for (int t = 0; t < 4; t++) f[t] = fp61::add(f2[0][t], fp61::mul(x[2][t], fp61::sub(f2[1][t], f2[0][t])));
        LA[e0] = f[2];
        if (m > 1) LA[(size_t)nE + e0] = f[3];
        uint64_t cur = f[3];
        uint64_t d1 = fp61::sub(f[3], f[2]);
        uint64_t d2 = fp61::sub(d1, fp61::sub(f[2], f[1]));
        const uint64_t d3 = fp61::sub(d2, fp61::sub(fp61::sub(f[2], f[1]), fp61::sub(f[1], f[0])));
#pragma unroll 1
        for (uint32_t t = 4; t <= s; t++) {
            d2 = fp61::add(d2, d3); d1 = fp61::add(d1, d2); cur = fp61::add(cur, d1);
            LA[(size_t)(t - 2) * nE + e0] = cur;
        }
    }
    cl_bar(4, CL_LT);
    uint64_t *cur = LA, *nxt = LB;
    uint32_t ne = nE;
#pragma unroll 1
    for (uint32_t k = 3; k < s; k++) {
        cl_line_wait(S, Rb + s + k + 1);                     // r2_k has been handed off
        if (lt < m) {                                        // l(t)_k, t = 2..s
            const uint64_t p = fp61::draw(seed, ctr0 + k), q = fp61::draw(seed, ctr0 + s + k);
            S.lpts[lt] = fp61::add(p, fp61::mul(lt + 2, fp61::sub(q, p)));
        }
        cl_bar(4, CL_LT);
        if (k < sb) {                                        // a level of the block's tree: one multiply per (node, t)
            const uint32_t lh = sb - k - 1, nh = 1u << lh;   // ne = 2 nh
#pragma unroll 1
            for (uint32_t it = lt; it < (m << lh); it += CL_LT) {
                const uint32_t t = it >> lh, u = it & (nh - 1);
                const ulonglong2 ab = *reinterpret_cast<const ulonglong2 *>(cur + (size_t)t * ne + 2 * u);
                nxt[(size_t)t * nh + u] = fold2(ab.x, ab.y, S.lpts[t]);
            }
            uint64_t *tmp = cur; cur = nxt; nxt = tmp;
            ne = nh;
        } else if (lt < m) {                                 // a block-index variable: the block's weight eq(block bits, l(t))
            cur[lt] = fp61::mul(cur[lt], fp61::chi((rank >> (k - sb)) & 1u, S.lpts[lt]));
        }
        cl_bar(4, CL_LT);
    }
    if (lt < m) cx.acc[lt] = cur[lt];
}

// After q[2..s] sit in cx.acc: warp 0 writes q[0..s] (if writer), draws tau, sets z <- l(tau), claim <- q(tau) by Lagrange
// interpolation on the nodes 0..s (denominators prepared in S.dk), ctr <- ctr0 + 2s + 1.  s <= 30.
__device__ __forceinline__ void cl_finish(uint32_t s, ClShared &S, uint32_t ctr0, uint64_t *tr_q, bool writer) {
    FusedCtx &cx = S.cx;
    const uint32_t k = threadIdx.x & 31;
    const uint64_t seed = cx.seed;
    const uint64_t r1k = k < s ? fp61::draw(seed, ctr0 + k) : 0, r2k = k < s ? fp61::draw(seed, ctr0 + s + k) : 0;
    uint64_t qk = 0;
    if (k <= s) {
        qk = k == 0 ? cx.v1 : (k == 1 ? cx.v2 : cx.acc[k - 2]);
        if (writer) tr_q[k] = qk;                            // the message q[0..s] is out before tau is used
    }
    const uint64_t qd = k <= s ? fp61::mul(qk, S.dk[k]) : 0;
    const uint64_t tau = fp61::draw(seed, ctr0 + 2 * s);
    const uint64_t f = k <= s ? fp61::sub(tau, k) : 1;
    uint64_t pre = f, suf = f;                               // prefix and suffix products of (tau - k) across the lanes
#pragma unroll
    for (uint32_t off = 1; off < 32; off <<= 1) {
        if (off > s) break;
        const uint64_t up = __shfl_up_sync(0xffffffffu, pre, off), dn = __shfl_down_sync(0xffffffffu, suf, off);
        if (k >= off) pre = fp61::mul(pre, up);
        if (k + off < 32) suf = fp61::mul(suf, dn);
    }
    const uint64_t pl = __shfl_up_sync(0xffffffffu, pre, 1), sr = __shfl_down_sync(0xffffffffu, suf, 1);
    const uint64_t num = fp61::mul(k ? pl : 1, k < 31 ? sr : 1);
    const uint64_t claim = warp_sum61(k <= s ? fp61::mul(qd, num) : 0);
    const uint64_t znew = k < s ? fold2(r1k, r2k, tau) : 0;
    if (k < s) cx.z[k] = znew;
    if (k == 0) { cx.claim = claim; cx.ctr = ctr0 + 2 * s + 1; }
}

// One persistent kernel for a run of consecutive layers, launched as ONE cluster.
__global__ void __launch_bounds__(CL_T, 1) k_cluster(ClArgs a) {
    extern __shared__ __align__(16) uint8_t cl_smem_raw[];
    ClShared &S = *reinterpret_cast<ClShared *>(cl_smem_raw);
    uint8_t *dyn = cl_smem_raw + ((sizeof(ClShared) + 15) & ~(size_t)15);
    FusedCtx &cx = S.cx;
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, rank = cl_rank();
    const bool linew = tid >= CL_GT && tid < CL_GT + CL_LT, trw = warp == (CL_GT + CL_LT) / 32, svc = warp == (CL_GT + CL_LT) / 32 + 1;
#ifdef VC_TRACE
    const bool trace_thread = rank == 0 && tid == 0;
    uint32_t trow[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    if (tid == 0 && rank == 0) { g_tr_stamps = a.stamps; g_tr_d = a.d; S.trn = 0; }
#endif
    {   // the plans of this launch's layers: one read from global memory, at the start
        const uint32_t nl = a.end - a.begin;
        constexpr uint32_t WC = sizeof(ClLayer) / 4, WL = sizeof(LayerPlan) / 4;
        for (uint32_t i = tid; i < nl * WC; i += CL_T)
            reinterpret_cast<uint32_t *>(&S.pl[i / WC].C)[i % WC] = reinterpret_cast<const uint32_t *>(a.cl + a.begin + i / WC)[i % WC];
        for (uint32_t i = tid; i < nl * WL; i += CL_T)
            reinterpret_cast<uint32_t *>(&S.pl[i / WL].Lp)[i % WL] = reinterpret_cast<const uint32_t *>(a.L + a.begin + i / WL)[i % WL];
        if (tid < nl) { S.pl[tid].Vb = a.L[a.begin + tid + 1].V; S.pl[tid].s = a.L[a.begin + tid + 1].log_n; }
    }
    if (a.begin == 0) {
        const uint32_t s0 = a.L[0].log_n;
        if (tid < s0) cx.z[tid] = fp61::draw(a.seed, tid);           // a2: z_0
        if (tid == 0) { cx.seed = a.seed; cx.ctr = s0; cx.claim = 0; }
    } else {
        if (tid < MAX_VARS) cx.z[tid] = a.st->z[tid];
        if (tid == 0) { cx.seed = a.seed; cx.ctr = a.st->ctr; cx.claim = a.st->claim; }
    }
    if (tid <= MAX_VARS) S.invfact[tid] = a.st->invfact[tid];
    build_pascal(S.pas, tid);
    if (tid == 0) {
        cx.epoch = a.st->bar_gen; cx.v1 = 0; cx.v2 = 0; cx.pad = 0;
        cl_mbar_init(&S.mb_rd[0], CL_C); cl_mbar_init(&S.mb_rd[1], CL_C);
        cl_mbar_init(&S.mb_end[0], 1); cl_mbar_init(&S.mb_end[1], 1);
        for (int k = 0; k < 8; k++) cl_mbar_init(&S.mb_dat[k], 1);
        cl_mbar_init(&S.mb_gat[0], 1); cl_mbar_init(&S.mb_gat[1], 1);
        cl_mbar_init(&S.mb_state, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (tid == 0) { S.rounds_done = 0; S.svc_done = 0; S.tr_done = 0; }
    __syncthreads();
    cl_sync_all();                                               // every CTA's mbarriers exist before anyone arrives on them
    if (svc) cl_svc_role(a, S, rank);
    else if (trw) { if (rank == 0) cl_tr_role(a, S); }
    else {
        constexpr uint32_t NM = CL_T - 64;                       // the threads of the layer loop: everyone but the two pipeline warps
        uint64_t *tr = a.tr;
        ClPhases php = {{0, 0}, {0, 0}, {0, 0, 0, 0, 0, 0, 0, 0}, {0, 0}, 0};
        uint32_t Rb = 0;
        ClPre pre; pre.layer = 0xffffffffu; pre.i1 = pre.i2 = 0; pre.t = VC_RELAY; pre.other = 0;
        for (uint32_t layer = a.begin; layer < a.end; layer++) {
            const ClLayer &C = S.pl[layer - a.begin].C;
            const uint32_t s = S.pl[layer - a.begin].s, A = C.A, lp = (layer - a.begin) & 1u;
            if (rank < A) {
                const uint32_t prevA = layer > a.begin ? S.pl[layer - 1 - a.begin].C.A : 0;
                if (pre.layer != layer) cl_fetch(a, S, dyn, layer, rank, pre);   // first layer of the launch, or a CTA that joins
                if (prevA && rank >= prevA) {                    // this CTA joins: (z, claim, ctr) come from CTA 0
                    if (tid == 0) cl_mbar_expect(&S.mb_state, (MAX_VARS + 2) * 8);
                    cl_mbar_wait(&S.mb_state, php.state);
                    php.state ^= 1u;
                    if (tid < MAX_VARS) cx.z[tid] = S.state_in[tid];
                    if (tid == 0) { cx.claim = S.state_in[MAX_VARS]; cx.ctr = S.state_in[MAX_VARS + 1]; }
                    cl_bar(5, NM);
                }
                if (rank == 0 && tid == 0) a.stamps[layer] = globaltimer_ns();
                CL_TRC(0);
                if (A > 1 && tid == 0) cl_mbar_expect(&S.mb_end[lp], A * (s - 1) * 8);
                const uint32_t ctr0 = (uint32_t)cx.ctr;
                const bool part = tid < C.ngt || (tid >= CL_GW && tid < CL_GW + C.nft);
                if (part) cl_rounds(a, S, dyn, layer, rank, Rb, php, pre);
                else {
                    if (linew) {
                        const uint32_t lt = tid - CL_GT;
                        if (lt <= s) {                           // the Lagrange denominators of the finish
                            const uint64_t dkv = fp61::mul(S.invfact[lt], S.invfact[s - lt]);
                            S.dk[lt] = ((s - lt) & 1u) ? fp61::neg(dkv) : dkv;
                        }
                        if (C.lmode == CL_LINE_STREAM || C.lmode == CL_LINE_DIRECT) cl_line_stream(a, S, dyn, layer, rank, Rb);
                    }
                    // the mbarrier phases this CTA went through, for threads that sat the rounds out
                    if (A > 1) { php.rd[0] ^= s & 1u; php.rd[1] ^= s & 1u; }
                    if (C.m[0] < s) php.gat[0] ^= 1u;
                    if (C.m[1] < s) php.gat[1] ^= 1u;
                }
                Rb += 2 * s;
                CL_TRC(1);
                cl_bar(5, NM);
                CL_TRC(2);
                if (C.lmode == CL_LINE_PASS) {                   // a7 as a separate pass (blocks too large to stream)
                    if (tid < 2 * s) {
                        const uint64_t r = fp61::draw(cx.seed, ctr0 + tid);
                        if (tid < s) cx.r1[tid] = r; else cx.r2[tid - s] = r;
                    }
                    cl_bar(5, NM);
                    if (tid < C.lthr) line_partials(S.pl[layer - a.begin].Vb, s, cx, S.pas, reinterpret_cast<uint64_t *>(dyn), rank, A, tid, C.lthr, C.ltb);
                    cl_bar(5, NM);
                }
                if (layer + 1 < a.end && rank < S.pl[layer + 1 - a.begin].C.A) cl_fetch(a, S, dyn, layer + 1, rank, pre);   // the next layer's loads travel during the finish
                if (A > 1) {                                     // the s-1 block values of every CTA go to all A CTAs
                    for (uint32_t i = tid; i < (s - 1) * A; i += NM) {
                        const uint32_t peer = i / (s - 1), k = i - peer * (s - 1);
                        cl_st_async(cl_mapa(cl_smem(&S.qin[lp][rank][k]), peer), cx.acc[k], cl_mapa(cl_smem(&S.mb_end[lp]), peer));
                    }
                    if (warp == 0) {
                        cl_mbar_wait(&S.mb_end[lp], php.end[lp]);
                        if (lane < s - 1) {
                            uint64_t sum = 0;
                            for (uint32_t c = 0; c < A; c++) sum = fp61::add(sum, S.qin[lp][c][lane]);
                            cx.acc[lane] = sum;
                        }
                        __syncwarp();
                    }
                    php.end[lp] ^= 1u;
                }
                CL_TRC(3);
                if (warp == 0) cl_finish(s, S, ctr0, tr + 6 * (size_t)s, rank == 0);
                cl_bar(5, NM);
                if (rank == 0 && layer + 1 < a.end && S.pl[layer + 1 - a.begin].C.A > A) {   // wider layer next: hand the state to the CTAs that join
                    const uint32_t An = S.pl[layer + 1 - a.begin].C.A;
                    for (uint32_t i = tid; i < (An - A) * (MAX_VARS + 2); i += NM) {
                        const uint32_t peer = A + i / (MAX_VARS + 2), k = i % (MAX_VARS + 2);
                        const uint64_t v = k < MAX_VARS ? cx.z[k] : (k == MAX_VARS ? cx.claim : cx.ctr);
                        cl_st_async(cl_mapa(cl_smem(&S.state_in[k]), peer), v, cl_mapa(cl_smem(&S.mb_state), peer));
                    }
                }
                CL_TRC(4);
                CL_TRC_ROW(1000u * layer + 999u);
            }
            tr += 7 * (size_t)s + 1;
        }
    }
    if (rank == 0 && tid == 0) a.stamps[a.end] = globaltimer_ns();
    __syncthreads();                                             // the pipeline warps have written the last transcript words
    if (rank == 0) {
        if (tid < MAX_VARS) a.st->z[tid] = cx.z[tid];
        if (tid == 0) { a.st->seed = cx.seed; a.st->ctr = cx.ctr; a.st->claim = cx.claim; a.st->bar_gen = cx.epoch; }
    }
#ifdef VC_TRACE
    if (rank == 0) {
        __syncthreads();
        uint32_t *out = reinterpret_cast<uint32_t *>(a.stamps + a.d + 1);
        if (tid == 0) out[0] = S.trn;
        for (uint32_t i = tid; i < S.trn * 8; i += CL_T) out[8 + i] = S.trc[i >> 3][i & 7];
    }
#endif
    cl_sync_all();                                           // no CTA leaves while a peer may still write into it
}

}  // namespace vc
