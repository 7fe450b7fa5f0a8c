// vc_fused.cu — kernel + host driver (load-time plan, launch) of the on-chip schedule (see vc_fused.cuh).
#include <algorithm>
#include <cstdio>
#include <new>
#include <cstdlib>
#include <vector>

#include "vc_circuit.hpp"
#include "vc_cluster.cuh"
#include "vc_fused_small.cuh"
#include "vc_fused_thin.cuh"
#include "vc_fused_wide.cuh"

namespace vc {

// MASK: which layer kinds this instantiation contains (1 narrow single-CTA, 2 thin, 4 wide).  The whole proof can run in
// the all-kinds kernel; when the layers of a circuit fall into few runs of {narrow, thin} and {wide}, each run is
// launched in the kernel that holds only its own code (the proof state travels through DevState, as it does between
// vc_prove_layer calls): the resident loop of the wide path then gets the registers of the kernel to itself.
template <int MASK>
__global__ void __launch_bounds__(FT, 1) k_fused(FusedArgs a) {
    extern __shared__ __align__(16) uint8_t smem[];
    FusedCtx &cx = *reinterpret_cast<FusedCtx *>(smem);
    uint64_t *invfact = reinterpret_cast<uint64_t *>(smem + F_INVFACT_OFF);        // 1/k!, k <= MAX_VARS
    uint32_t *pas = reinterpret_cast<uint32_t *>(smem + F_PASCAL_OFF);             // C(n,k), n,k < 32
    uint8_t *dyn = smem + F_FIXED_BYTES;
    const uint32_t tid = threadIdx.x;
#ifdef VC_TRACE
    if (tid == 0) { g_tr_stamps = a.stamps; g_tr_d = a.d; }
#endif
    // ---- load (or start) the proof state
    if (a.begin == 0) {
        const uint32_t s0 = a.L[0].log_n;
        if (tid < s0) cx.z[tid] = fp61::draw(a.seed, tid);      // a2: z_0
        if (tid == 0) { cx.seed = a.seed; cx.ctr = s0; cx.claim = 0; }
    } else {
        if (tid < MAX_VARS) cx.z[tid] = a.st->z[tid];
        if (tid == 0) { cx.seed = a.seed; cx.ctr = a.st->ctr; cx.claim = a.st->claim; }
    }
    if (tid <= MAX_VARS) invfact[tid] = a.st->invfact[tid];
    build_pascal(pas, tid);
#ifdef VC_POISON                                   // debug build: uninitialised shared-memory reads become loud
    {
        uint32_t dsz;
        asm volatile("mov.u32 %0, %%dynamic_smem_size;" : "=r"(dsz));
        for (uint32_t i = tid; i < (dsz - (uint32_t)F_FIXED_BYTES) / 8; i += FT) reinterpret_cast<uint64_t *>(dyn)[i] = 0xDEADBEEFDEADBEEFull;
        if (tid < 128) cx.red[tid] = 0xDEADBEEFDEADBEEFull;
        if (tid < MAX_VARS) cx.acc[tid] = 0xDEADBEEFDEADBEEFull;
    }
#endif
    if (tid == 0) { cx.epoch = a.st->bar_gen; cx.v1 = 0; cx.v2 = 0; cx.pad = 0; }
    __syncthreads();
    uint64_t *tr = a.tr;
    bool handoff = false;                         // CTA 0 ran narrow layers alone: publish its state first
    for (uint32_t layer = a.begin; layer < a.end; layer++) {
        const uint32_t s = a.L[layer + 1].log_n;
        if (blockIdx.x == 0 && tid == 0) a.stamps[layer] = globaltimer_ns();
        VC_TR(100 + layer);
        if (tid < sizeof(WireRule) / 4) reinterpret_cast<uint32_t *>(&cx.wrule)[tid] = reinterpret_cast<const uint32_t *>(&a.L[layer].rule)[tid];
        __syncthreads();
        if (a.L[layer].kind == 0) {
            if (MASK & 1) { if (blockIdx.x == 0) small_layer(a, cx, invfact, pas, dyn, layer, tr); }
            handoff = true;
        } else {
            if (handoff) {
                if (blockIdx.x == 0) {
                    if (tid < MAX_VARS) a.st->z[tid] = cx.z[tid];
                    if (tid == 0) { a.st->ctr = cx.ctr; a.st->claim = cx.claim; }
                }
                grid_allreduce(cx, a, 0, true);
                if (blockIdx.x != 0) {
                    if (tid < MAX_VARS) cx.z[tid] = __ldcg(&a.st->z[tid]);
                    if (tid == 0) { cx.ctr = __ldcg(&a.st->ctr); cx.claim = __ldcg(&a.st->claim); }
                }
                __syncthreads();
                handoff = false;
            }
            if (a.L[layer].thin) {
                if (MASK & 2) {
                    if (a.L[layer].thin == 4) thin_layer<4>(a, cx, invfact, pas, dyn, layer, tr);
                    else thin_layer<1>(a, cx, invfact, pas, dyn, layer, tr);
                }
            } else if (MASK & 4) wide_layer(a, cx, invfact, pas, dyn, layer, tr);
        }
        tr += 7 * (size_t)s + 1;
    }
    // ---- leave the state for the next call
    if (blockIdx.x == 0 && tid == 0) a.stamps[a.end] = globaltimer_ns();
    if (blockIdx.x == 0) {
        if (tid < MAX_VARS) a.st->z[tid] = cx.z[tid];
        if (tid == 0) { a.st->seed = cx.seed; a.st->ctr = cx.ctr; a.st->claim = cx.claim; a.st->bar_gen = cx.epoch; }
    }
}

// ---- a1 in one launch: V_d <- input (checked canonical), then V_i[g] = f_type(V_{i+1}[in1[g]], V_{i+1}[in2[g]]) for
// i = d-1..0 (all gates of a layer in parallel, layer after layer).  Grid-wide layers are separated by a
// counter rendezvous; once the remaining layers are narrow CTA 0 finishes them alone behind block barriers, with the
// values in shared memory and the next layer's records fetched ahead.
constexpr int EVAL_T = 1024;
constexpr uint32_t EVAL_NARROW_LOG = 11;
__device__ __forceinline__ void eval_grid_barrier(unsigned int *cnt, uint32_t &gen) {
    __syncthreads();
    if (threadIdx.x == 0) {
        gen++;
        __threadfence();
        asm volatile("red.relaxed.gpu.global.add.u32 [%0], 1;" ::"l"(cnt) : "memory");
        const unsigned int want = gen * gridDim.x;
        unsigned int v;
        do { asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(cnt) : "memory"); } while (v < want);
    }
    __syncthreads();
}
// top: the first layer evaluated here is d-1, the last is `top` (0; 1 when layer 0 is the sum gate, which has its own kernel).
// loc_bl > 0: layers d-1 .. loc_top have block-local wiring (tree: 2g, 2g+1; self: g, g; one gate type each), so a block of
// 2^loc_bl inputs determines its own share of every one of them: a CTA checks and copies its inputs, then runs up the
// layers in shared memory (every V_i is still written out for the prover) with block barriers only; the grid meets once,
// after the local run, instead of once per layer.
#ifndef VC_EVAL_LOC_LOG
#define VC_EVAL_LOC_LOG 13
#endif
constexpr int EVAL_LOC_MAX = 32;                       // layers of a local run at most
constexpr uint32_t EVAL_LOC_LOG = VC_EVAL_LOC_LOG;                   // inputs per block of the local run (two tables of 2^13 words: one wave of 128 blocks at n = 2^20)
__global__ void __launch_bounds__(EVAL_T, 1) k_eval_all(const LayerPlan *L, uint32_t d, const uint64_t *in, uint64_t *out0,
                                                          DevState *st, int top, uint32_t loc_bl, int loc_top) {
    unsigned int *cnt = &st->bar_count;              // zeroed together with the status word when vc_evaluate is enqueued
    const uint32_t tid = threadIdx.x, G = gridDim.x, b = blockIdx.x;
    uint32_t gen = 0;
    extern __shared__ __align__(16) uint64_t ev_sm[];   // the narrow tail / the local run: two value tables of 2^(EVAL_NARROW_LOG+1) words
    int i = (int)d - 1;
    if (loc_bl) {
        uint64_t *Vd = const_cast<uint64_t *>(L[d].V);
        const uint32_t nblk = 1u << (L[d].log_n - loc_bl), B = 1u << loc_bl;
        unsigned bad = 0;
        // the plans of the local layers sit in global memory: one fetch per kernel, not one dependent L2 round trip per layer
        __shared__ uint64_t *s_V[EVAL_LOC_MAX];
        __shared__ uint32_t s_tree[EVAL_LOC_MAX], s_t0[EVAL_LOC_MAX];
        if (tid < (uint32_t)((int)d - loc_top)) {
            const LayerPlan &Lp = L[(int)d - 1 - (int)tid];
            s_V[tid] = const_cast<uint64_t *>(Lp.V); s_tree[tid] = Lp.wiring == W_TREE; s_t0[tid] = Lp.type0;
        }
        __syncthreads();
        for (uint32_t blk = b; blk < nblk; blk += G) {
            uint64_t *cur = ev_sm, *nxt = ev_sm + B;
            {   // all of the block's input loads in flight before the first use (B / EVAL_T <= 8 words per thread, 16 B each)
                constexpr uint32_t NV = (1u << EVAL_LOC_LOG) / (2 * EVAL_T);
                const ulonglong2 *in2 = reinterpret_cast<const ulonglong2 *>(in + (size_t)blk * B);
                ulonglong2 *Vd2 = reinterpret_cast<ulonglong2 *>(Vd + (size_t)blk * B), *cur2 = reinterpret_cast<ulonglong2 *>(cur);
                ulonglong2 w[NV];
#pragma unroll
                for (uint32_t k = 0; k < NV; k++) w[k] = in2[k * EVAL_T + tid];
#pragma unroll
                for (uint32_t k = 0; k < NV; k++) {
                    bad |= (w[k].x >= fp61::P) | (w[k].y >= fp61::P);
                    Vd2[k * EVAL_T + tid] = w[k];
                    cur2[k * EVAL_T + tid] = w[k];
                }
            }
            __syncthreads();
            uint32_t share = B;                          // this block's entries of the layer below
            for (int l = (int)d - 1; l >= loc_top; l--) {
                const bool tree = s_tree[(int)d - 1 - l] != 0;
                const uint32_t t0 = s_t0[(int)d - 1 - l];
                if (tree) share >>= 1;
                uint64_t *Vo = s_V[(int)d - 1 - l] + (size_t)blk * share;
                for (uint32_t g = tid; g < share; g += EVAL_T) {
                    const uint64_t v = tree ? gate_f(t0, cur[2 * g], cur[2 * g + 1]) : gate_f(t0, cur[g], cur[g]);
                    nxt[g] = v; Vo[g] = v;
                    if (l == 0 && out0) out0[(size_t)blk * share + g] = v;
                }
                __syncthreads();
                uint64_t *t = cur; cur = nxt; nxt = t;
            }
        }
        if (bad) atomicOr(&st->flags, 1u);
        i = loc_top - 1;
    } else
    {
        uint64_t *Vd = const_cast<uint64_t *>(L[d].V);
        const uint64_t n = 1ull << L[d].log_n;
        unsigned bad = 0;
        for (uint64_t i = b * (uint64_t)EVAL_T + tid; i < n; i += (uint64_t)G * EVAL_T) {
            const uint64_t w = in[i];
            bad |= (w >= fp61::P);
            Vd[i] = w;
        }
        if (bad) atomicOr(&st->flags, 1u);
    }
    for (; i >= top; i--) {                       // grid-wide layers, separated by a counter rendezvous
        if (L[i].log_n <= EVAL_NARROW_LOG && L[i + 1].log_n <= EVAL_NARROW_LOG + 1) break;
        const uint32_t n = 1u << L[i].log_n;
        const Wires wr(L[i]);
        const uint64_t *Vb = L[i + 1].V;
        uint64_t *Vo = const_cast<uint64_t *>(L[i].V);
        eval_grid_barrier(cnt, gen);
        for (uint32_t g = b * EVAL_T + tid; g < n; g += G * EVAL_T) {
            uint32_t i1, i2, t;
            wr.get(g, i1, i2, t);
            const uint64_t v = gate_f(t, __ldcg(Vb + i1), __ldcg(Vb + i2));
            Vo[g] = v;
            if (i == 0 && out0) out0[g] = v;
        }
    }
    if (i < top) return;
    // ---- CTA 0 finishes the narrow layers alone: values ping-pong in shared memory (every V_i is still written out
    // for the prover), and the records of the next layer are fetched before the barrier that ends the current one
    eval_grid_barrier(cnt, gen);
    if (b != 0) return;
    constexpr uint32_t TW = 2u << EVAL_NARROW_LOG, NG = (1u << EVAL_NARROW_LOG) / EVAL_T;   // table words; gates per thread
    uint64_t *cur = ev_sm, *nxt = ev_sm + TW;
    {
        const uint64_t *Vb = L[i + 1].V;
        for (uint32_t u = tid; u < (1u << L[i + 1].log_n); u += EVAL_T) cur[u] = __ldcg(Vb + u);
    }
    uint32_t rt[NG], ra[NG], rb[NG];
    auto fetch = [&](int layer) {
        const uint32_t n = 1u << L[layer].log_n;
#pragma unroll
        for (uint32_t k = 0; k < NG; k++) {
            const uint32_t g = k * EVAL_T + tid;
            if (g < n) Wires(L[layer]).get(g, ra[k], rb[k], rt[k]);
        }
    };
    fetch(i);
    __syncthreads();
    for (; i >= top; i--) {
        const uint32_t n = 1u << L[i].log_n;
        uint64_t *Vo = const_cast<uint64_t *>(L[i].V);
#pragma unroll
        for (uint32_t k = 0; k < NG; k++) {
            const uint32_t g = k * EVAL_T + tid;
            if (g < n) {
                const uint64_t v = gate_f(rt[k], cur[ra[k]], cur[rb[k]]);
                nxt[g] = v; Vo[g] = v;
                if (i == 0 && out0) out0[g] = v;
            }
        }
        if (i > top) fetch(i - 1);
        __syncthreads();
        uint64_t *t = cur; cur = nxt; nxt = t;
    }
}

constexpr size_t EVAL_SMEM = 2 * (size_t)((2u << EVAL_NARROW_LOG) > (1u << EVAL_LOC_LOG) ? (2u << EVAL_NARROW_LOG) : (1u << EVAL_LOC_LOG)) * 8;

constexpr size_t F_SMEM_MAX = 227 * 1024;
constexpr size_t F_MAX_RUNS = 8;                   // more runs of layer kinds than this: the all-kinds kernel, one launch

struct FusedHost {
    LayerPlan *d_plan = nullptr;
    CtaPlan *d_cta = nullptr;
    unsigned long long *d_slots = nullptr;
    uint64_t *d_stamps = nullptr, *d_C = nullptr, *d_Tg = nullptr;
    bool eval_ok = false;
    uint32_t eval_loc_bl = 0;                      // k_eval_all's block-local run: log2 inputs per block (0: none), last local layer
    int eval_loc_top = 0;
    std::vector<int> group;                        // per layer: 1 narrow, 2 thin, 4 wide (which k_fused instantiation holds its code), 8 = the cluster engine
    int grid = 0;
    size_t smem = 0;
    ClLayer *d_cl = nullptr;                       // the cluster engine's plans (vc_cluster.cuh)
    int csize = 0;                                 // CTAs per cluster (0: engine unavailable)
    bool single_kernel = false;                    // VC_SINGLE_KERNEL=1 in the environment at load: always the all-kinds kernel (A/B measurements)
    size_t cl_smem = 0;
};
static std::vector<std::pair<const vc_circuit *, FusedHost *>> g_fused;   // heap entries: pointers handed out by find() stay valid
static void release(FusedHost *f) {
    if (!f) return;
    cudaFree(f->d_plan); cudaFree(f->d_cta); cudaFree(f->d_slots); cudaFree(f->d_stamps); cudaFree(f->d_C); cudaFree(f->d_Tg); cudaFree(f->d_cl);
    delete f;
}

static FusedHost *find(const vc_circuit *c) {
    std::lock_guard<std::mutex> lk(g_registry_mutex);
    for (auto &p : g_fused) if (p.first == c) return p.second;
    return nullptr;
}

// ---- the load-time plan: how each layer is partitioned over the CTAs, which table mode each phase uses and where
// its buffers sit in shared memory.  Pure index bookkeeping on the host copy of the records.
static void plan_layer(const vc_circuit *c, uint32_t i, int G, LayerPlan &lp, std::vector<CtaPlan> &cta, size_t &smem_need) {
    const uint32_t si = c->logs[i], s = c->logs[i + 1];
    const uint64_t n = 1ull << si;
    lp.log_n = si;
    lp.kind = (si <= (uint32_t)F_SMALL_N_LOG && s <= (uint32_t)F_SMALL_T_LOG) ? 0 : 1;
    lp.has_relay = 0;
    for (uint8_t t : c->h_type[i]) if (t == VC_RELAY) { lp.has_relay = 1; break; }
    lp.thin = 0; lp.resident = 0; lp.cap = 0; lp.mode[0] = lp.mode[1] = F_MODE_GLOBAL; lp.K[0] = lp.K[1] = 0;
    lp.xw = lp.yw = 0; lp.off_tab = lp.off_scr = lp.off_commit = 0;
    if (lp.kind == 0) { smem_need = std::max(smem_need, F_FIXED_BYTES + F_SMALL_BYTES); return; }
    // gates in units of 32, spread evenly over the CTAs
    const uint64_t U = (n + 31) / 32;
    uint64_t ngmax = 0;
    cta.assign(G, CtaPlan{});
    const uint32_t K = s > (uint32_t)F_TLOG ? s - F_TLOG : 0;
    uint64_t nbmax[2] = {0, 0};
    for (int b = 0; b < G; b++) {
        const uint64_t g0 = std::min<uint64_t>(n, 32 * ((uint64_t)b * U / G)), g1 = std::min<uint64_t>(n, 32 * ((uint64_t)(b + 1) * U / G));
        cta[b].g0 = (uint32_t)g0; cta[b].g1 = (uint32_t)g1;
        ngmax = std::max(ngmax, g1 - g0);
        for (int ph = 0; ph < 2; ph++) {
            const std::vector<uint32_t> &idx = ph == 0 ? c->h_in1[i] : c->h_in2[i];
            uint32_t lo = 0xffffffffu, hi = 0;
            for (uint64_t g = g0; g < g1; g++) { lo = std::min(lo, idx[g]); hi = std::max(hi, idx[g]); }
            if (g1 > g0) { cta[b].blo[ph] = lo >> K; cta[b].nb[ph] = (hi >> K) - (lo >> K) + 1; }
            nbmax[ph] = std::max<uint64_t>(nbmax[ph], cta[b].nb[ph]);
        }
    }
    // level K-1 published from the slices: CTAs in order take the entries of their slice nobody before them took; that
    // works when the slices cover the whole level without a gap (regular wiring), else the owners compute their entries from V
    bool cover[2] = {K >= 2, K >= 2};
    for (int ph = 0; ph < 2; ph++) {
        const uint64_t E = 1ull << (s - K + 1);
        uint64_t next = 0;
        for (int b = 0; b < G && cover[ph]; b++) {
            cta[b].own_lo[ph] = cta[b].own_n[ph] = 0;
            if (cta[b].g1 == cta[b].g0) continue;
            const uint64_t lo = 2ull * cta[b].blo[ph], hi = 2ull * ((uint64_t)cta[b].blo[ph] + cta[b].nb[ph]);
            if (lo > next) { cover[ph] = false; break; }
            if (hi > next) { cta[b].own_lo[ph] = (uint32_t)next; cta[b].own_n[ph] = (uint32_t)(hi - next); next = hi; }
        }
        if (next != E) cover[ph] = false;
        if (getenv("VC_NO_PUB_SLICE")) cover[ph] = false;
    }
    const size_t cap = (size_t)((ngmax + FT - 1) / FT) * FT;
    const size_t state = cap * 20;
    // fold buffers: odd levels in X, even levels in Y; slices exist for levels 1..K-1
    auto buf_words = [&](int ph, size_t &xw, size_t &yw) {
        xw = (size_t)1 << (s >= 1 ? std::min<uint32_t>(s - 1, F_TLOG) : 0);
        yw = (size_t)1 << (s >= 2 ? std::min<uint32_t>(s - 2, F_TLOG) : 0);
        if (K >= 2) xw = std::max(xw, (size_t)nbmax[ph] << (K - 1));
        if (K >= 3) yw = std::max(yw, (size_t)nbmax[ph] << (K - 2));
    };
    const size_t scr_words = (1u << F_EQLOG) + 64;
    bool slice_ok[2];
    for (int ph = 0; ph < 2; ph++) slice_ok[ph] = K <= (uint32_t)F_EQLOG + 1;   // the owner's eq table covers K-1 <= 10 variables
    if (ngmax <= F_WORKERS && slice_ok[0] && slice_ok[1]) {     // thin layer: gate in registers, commit buffers instead of state
        size_t xw[2], yw[2];
        buf_words(0, xw[0], yw[0]); buf_words(1, xw[1], yw[1]);
        size_t X = std::max<size_t>(1024, std::max(xw[0], xw[1])), Y = std::max<size_t>(1024, std::max(yw[0], yw[1]));
        X = (X + 1) & ~(size_t)1; Y = (Y + 1) & ~(size_t)1;
        const size_t tabw = std::max<size_t>(X + Y, 4u << F_EQLOG);
        const size_t total = std::max(F_FIXED_BYTES + F_THIN_COMMIT_BYTES + tabw * 8 + scr_words * 8,
                                      F_FIXED_BYTES + fused_line_words(s, FT) * 8);
        if (total <= F_SMEM_MAX) {
            lp.thin = ngmax <= F_WORKERS / 4 ? 4 : 1;        // lanes per gate
            lp.cap = (uint32_t)cap;
            for (int ph = 0; ph < 2; ph++) { lp.mode[ph] = F_MODE_SLICE; lp.K[ph] = K; lp.pub_slice[ph] = cover[ph] ? 1u : 0u; }
            lp.xw = (uint32_t)X; lp.yw = (uint32_t)Y;
            lp.off_tab = (uint32_t)F_THIN_COMMIT_BYTES;
            lp.off_scr = (uint32_t)(F_THIN_COMMIT_BYTES + tabw * 8);
            smem_need = std::max(smem_need, total);
            return;
        }
    }
    // try: resident state + slices, then non-resident + slices, then drop the larger slice, ...
    for (int attempt = 0; attempt < 6; attempt++) {
        const bool res = attempt < 3;
        const int drop = attempt % 3;            // 0: both phases sliced, 1: drop the larger, 2: drop both
        bool use[2] = {slice_ok[0], slice_ok[1]};
        size_t xw[2], yw[2];
        buf_words(0, xw[0], yw[0]); buf_words(1, xw[1], yw[1]);
        if (drop >= 1) { const int big = (xw[0] + yw[0] >= xw[1] + yw[1]) ? 0 : 1; use[big] = false; }
        if (drop >= 2) use[0] = use[1] = false;
        size_t X = 1024, Y = 1024;
        for (int ph = 0; ph < 2; ph++) if (use[ph]) { X = std::max(X, xw[ph]); Y = std::max(Y, yw[ph]); }
        X = (X + 1) & ~(size_t)1; Y = (Y + 1) & ~(size_t)1;
        const size_t tabw = std::max<size_t>(X + Y, 4u << F_EQLOG);
        const size_t st_bytes = res ? state : 0;
        const size_t commit_bytes = (size_t)FT * 32;
        const size_t total = std::max(F_FIXED_BYTES + st_bytes + tabw * 8 + scr_words * 8 + commit_bytes,
                                      F_FIXED_BYTES + fused_line_words(s, FT) * 8);   // the line restriction reuses the whole region
        if (total > F_SMEM_MAX) continue;
        lp.resident = res ? 1 : 0;
        lp.cap = (uint32_t)cap;
        for (int ph = 0; ph < 2; ph++) { lp.mode[ph] = use[ph] ? F_MODE_SLICE : F_MODE_GLOBAL; lp.K[ph] = K; lp.pub_slice[ph] = (use[ph] && cover[ph]) ? 1u : 0u; }
        lp.xw = (uint32_t)X; lp.yw = (uint32_t)Y;
        lp.off_tab = (uint32_t)st_bytes;
        lp.off_scr = (uint32_t)(st_bytes + tabw * 8);
        lp.off_commit = (uint32_t)(st_bytes + tabw * 8 + scr_words * 8);
        smem_need = std::max(smem_need, total);
        return;
    }
    // unreachable: the last attempt (non-resident, no slices) needs only the fixed buffers
}

// ---- the cluster engine's load-time plan (vc_cluster.cuh): how many CTAs take a layer, which block of V_{i+1} each
// CTA's gates read in each phase, how the line restriction is blocked.  Index bookkeeping on the host copy of the records.
static size_t cl_line_words(uint32_t s, uint32_t tb) {
    const size_t sp = s < 3 ? 3 : s, P = tb + 4, NB = (size_t)1 << tb;
    return (((s + 1) * sp + 1) & ~(size_t)1) + NB * P + (NB * P + 1) / 2 + 1 + 64 + 8;
}
static bool plan_cluster_layer(const vc_circuit *c, uint32_t i, int csize, ClLayer &cl, size_t &dyn_bytes) {
    static const int target_gpc = getenv("VC_CL_GPC") ? atoi(getenv("VC_CL_GPC")) : 128;
    static const int single_max = getenv("VC_CL_SINGLE") ? atoi(getenv("VC_CL_SINGLE")) : 256;
    const uint32_t si = c->logs[i], s = c->logs[i + 1];
    cl = ClLayer{};
    if (si > CL_MAX_N || s > CL_MAX_S) return false;
    const uint32_t n = 1u << si;
    uint32_t A = 1;
    if ((int)n > single_max) { while (A < (uint32_t)csize && n / A > (uint32_t)target_gpc) A <<= 1; }
    while (n / A > (uint32_t)CL_GW) { if (A >= (uint32_t)csize) return false; A <<= 1; }
    if (A > n) A = n;
    const uint32_t gpc = n / A;
    uint32_t mmax = 1;
    for (int ph = 0; ph < 2; ph++) {
        const std::vector<uint32_t> &idx = ph == 0 ? c->h_in1[i] : c->h_in2[i];
        uint32_t m = 1, blk[CL_C] = {0};
        for (uint32_t b = 0; b < A; b++) {
            uint32_t lo = 0xffffffffu, hi = 0;
            for (uint32_t g = b * gpc; g < (b + 1) * gpc; g++) { lo = std::min(lo, idx[g]); hi = std::max(hi, idx[g]); }
            while ((lo >> m) != (hi >> m)) m++;
            blk[b] = lo;
        }
        bool sliced = A > 1 && m < s && (1u << (s - m)) == A;
        if (sliced) {                            // the A blocks must be the A distinct aligned blocks of the table
            uint32_t seen = 0;
            for (uint32_t b = 0; b < A; b++) seen |= 1u << (blk[b] >> m);
            sliced = seen == (A == 32 ? 0xffffffffu : (1u << A) - 1);
        }
        if (!sliced) m = s;
        if (m > CL_MAX_M) return false;
        cl.m[ph] = m;
        for (uint32_t b = 0; b < A; b++) cl.blk[ph][b] = sliced ? blk[b] >> m : 0;
        mmax = std::max(mmax, m);
    }
    cl.A = A; cl.gpc = gpc;
    cl.ngt = (gpc + 31) & ~31u;
    uint32_t nft = std::min<uint32_t>(CL_FW, std::max<uint32_t>(32, 1u << (mmax - 1)));
    if (si > 6 && cl.ngt + nft < 192) nft = 192 - cl.ngt;
    cl.nft = (nft + 31) & ~31u;
    uint32_t la = 0; while ((1u << la) < A) la++;
    if (s < la) return false;
    cl.sb = s - la;
    const size_t tabw = std::max<size_t>((size_t)1 << mmax, 64) + std::max<size_t>((size_t)1 << (mmax - 1), 64) +
                        std::max<size_t>((size_t)1 << cl.m[1], 64);       // X, Y and the phase-2 level 0
    cl.off_line = (uint32_t)(tabw * 8);
    size_t need = tabw * 8;
    cl.ltb = 0; cl.lthr = 32;
    if (s == 1) cl.lmode = CL_LINE_NONE;
    else if (cl.sb < 3) cl.lmode = CL_LINE_DIRECT;
    else {
        const size_t nE = (size_t)1 << (cl.sb - 3), lw = nE * (s - 1) + std::max<size_t>(nE / 2, 1) * (s - 1) + 2;
        if (lw * 8 <= 72 * 1024) { cl.lmode = CL_LINE_STREAM; need += lw * 8; }
        else {
            // a separate pass after the rounds: blocks of 2^tb threads x 8 words, at least one block per active CTA when the table allows it
            cl.lmode = CL_LINE_PASS;
            const uint32_t sp = s < 3 ? 3 : s;
            uint32_t tb = fused_line_tb(s, CL_GT);
            const uint32_t cap = sp - 3 > la ? sp - 3 - la : 0;
            tb = std::min(tb, cap);
            cl.ltb = tb;
            cl.lthr = std::max<uint32_t>(32, 1u << tb);
            need = std::max(need, cl_line_words(s, tb) * 8);
        }
    }
    dyn_bytes = std::max(dyn_bytes, need);
    return true;
}

static cudaError_t launch_cluster(const ClArgs &a, int csize, size_t smem, cudaStream_t st) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(csize); cfg.blockDim = dim3(CL_T); cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = csize; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, k_cluster, a);
}

static int fused_init_impl(vc_circuit *c, FusedHost &fh);
int fused_init(vc_circuit *c) {
    if (!c->coop_ok) return VC_OK;
    FusedHost *fh = new (std::nothrow) FusedHost();
    if (!fh) return VC_ERR_NOMEM;
    const int rc = fused_init_impl(c, *fh);
    if (rc != VC_OK || fh->grid == 0) { release(fh); return rc; }     // every partial allocation is returned; grid == 0: no fused schedule on this device
    std::lock_guard<std::mutex> lk(g_registry_mutex);
    g_fused.emplace_back(c, fh);
    return VC_OK;
}
static int fused_init_impl(vc_circuit *c, FusedHost &fh) {
    fh.grid = c->sm_count;
    std::vector<LayerPlan> h(c->d + 1);
    std::vector<CtaPlan> all_cta;
    std::vector<size_t> cta_off(c->d + 1, (size_t)-1);
    size_t smem_need = F_FIXED_BYTES + F_SMALL_BYTES;
    for (uint32_t i = 0; i <= c->d; i++) {
        LayerPlan &lp = h[i];
        lp = LayerPlan{};
        lp.type = i < c->d ? c->d_type[i] : nullptr;
        lp.in1 = i < c->d ? c->d_in1[i] : nullptr;
        lp.in2 = i < c->d ? c->d_in2[i] : nullptr;
        lp.V = c->d_V[i];
        lp.log_n = c->logs[i];
        lp.wiring = i < c->d ? c->wiring[i] : W_GENERIC;
        if (i < c->d) lp.rule = c->wrule[i];
        lp.type0 = i < c->d ? c->h_type[i][0] : 0;
        if (i < c->d && !(i == 0 && c->sum_out)) {       // the sum gate is not a fan-in-two layer: vc_sum.cuh proves it
            std::vector<CtaPlan> cta;
            plan_layer(c, i, fh.grid, lp, cta, smem_need);
            if (lp.kind == 1) { cta_off[i] = all_cta.size(); all_cta.insert(all_cta.end(), cta.begin(), cta.end()); }
        }
    }
    fh.smem = smem_need;
    if (cudaFuncSetAttribute(k_fused<7>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)F_SMEM_MAX) != cudaSuccess ||
        cudaFuncSetAttribute(k_fused<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)F_SMEM_MAX) != cudaSuccess ||
        cudaFuncSetAttribute(k_fused<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)F_SMEM_MAX) != cudaSuccess ||
        cudaFuncSetAttribute(k_fused<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)F_SMEM_MAX) != cudaSuccess) {
        (void)cudaGetLastError();
        fh.grid = 0;
        return VC_OK;                                // no fused schedule on this device; streaming still works
    }
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_fused<7>, FT, fh.smem) != cudaSuccess || per_sm < 1) {
        (void)cudaGetLastError();
        fh.grid = 0;
        return VC_OK;
    }
    uint64_t max_gates = 1;
    for (uint32_t i = 0; i < c->d; i++) max_gates = std::max<uint64_t>(max_gates, 1ull << c->logs[i]);
    if (cudaMalloc(&fh.d_plan, h.size() * sizeof(LayerPlan)) != cudaSuccess) return VC_ERR_NOMEM;
    if (cudaMalloc(&fh.d_cta, std::max<size_t>(all_cta.size(), 1) * sizeof(CtaPlan)) != cudaSuccess) return VC_ERR_NOMEM;
    if (cudaMalloc(&fh.d_slots, (size_t)F_RING * F_SLOT_WORDS * 8) != cudaSuccess) return VC_ERR_NOMEM;
    if (cudaMalloc(&fh.d_stamps, (size_t)(c->d + 1 + F_TRACE_WORDS) * 8) != cudaSuccess) return VC_ERR_NOMEM;
    if (cudaMalloc(&fh.d_C, max_gates * 8) != cudaSuccess) return VC_ERR_NOMEM;
    if (cudaMalloc(&fh.d_Tg, (size_t)(2u << F_TLOG) * 8) != cudaSuccess) return VC_ERR_NOMEM;
    {   // the one-launch evaluation needs: a co-resident grid, and narrow layers only at the output end
        int eper = 0;
        bool ok = cudaFuncSetAttribute(k_eval_all, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)EVAL_SMEM) == cudaSuccess &&
                  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&eper, k_eval_all, EVAL_T, EVAL_SMEM) == cudaSuccess && eper >= 1;
        bool seen_narrow = false;
        for (int i = (int)c->d - 1; i >= (int)c->first_pair_layer() && ok; i--) {
            const bool narrow = c->logs[i] <= EVAL_NARROW_LOG && c->logs[i + 1] <= EVAL_NARROW_LOG + 1;
            if (seen_narrow && !narrow) ok = false;
            seen_narrow = seen_narrow || narrow;
        }
        (void)cudaGetLastError();
        fh.eval_ok = ok;
        // the block-local run: layers d-1, d-2, ... while the wiring is tree (exactly half the layer below) or self (same size)
        // and a block of 2^EVAL_LOC_LOG inputs still owns at least one gate; worth it from three layers on
        if (ok && c->log_input > EVAL_LOC_LOG && !getenv("VC_NO_EVAL_LOCAL")) {
            uint32_t share_log = EVAL_LOC_LOG;
            int l = (int)c->d - 1;
            for (; l >= (int)c->first_pair_layer() && (int)c->d - 1 - l < EVAL_LOC_MAX; l--) {
                const uint32_t w = c->wiring[l];
                if (w == 1 && c->logs[l] + 1 == c->logs[l + 1] && share_log > 0) share_log--;
                else if (!(w == 2 && c->logs[l] == c->logs[l + 1])) break;
            }
            if ((int)c->d - 1 - l >= 3) { fh.eval_loc_bl = EVAL_LOC_LOG; fh.eval_loc_top = l + 1; }
        }
    }
    for (uint32_t i = 0; i < c->d; i++) h[i].cta = cta_off[i] == (size_t)-1 ? nullptr : fh.d_cta + cta_off[i];
    fh.group.resize(c->d);
    for (uint32_t i = 0; i < c->d; i++) fh.group[i] = h[i].kind == 0 ? 1 : (h[i].thin ? 2 : 4);
    if (c->sum_out) fh.group[0] = 0;
    if (const char *e = getenv("VC_SINGLE_KERNEL")) fh.single_kernel = e[0] == '1';
    {   // the cluster engine takes every layer it can plan (VC_NO_CLUSTER=1: never, for A/B measurements)
        const char *nc = getenv("VC_NO_CLUSTER");
        std::vector<ClLayer> hc(c->d);
        size_t dyn = 0;
        const size_t fixed = (sizeof(ClShared) + 15) & ~(size_t)15;
        int csize = 0;
        if (!(nc && nc[0] == '1') && !fh.single_kernel &&
            cudaFuncSetAttribute(k_cluster, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) == cudaSuccess &&
            cudaFuncSetAttribute(k_cluster, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)F_SMEM_MAX) == cudaSuccess) {
            for (int cs : {CL_C, CL_C / 2}) {
                cudaLaunchConfig_t cfg = {};
                cfg.gridDim = dim3(cs); cfg.blockDim = dim3(CL_T); cfg.dynamicSmemBytes = F_SMEM_MAX;
                cudaLaunchAttribute at[1];
                at[0].id = cudaLaunchAttributeClusterDimension;
                at[0].val.clusterDim.x = cs; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
                cfg.attrs = at; cfg.numAttrs = 1;
                int ncl = 0;
                if (cudaOccupancyMaxActiveClusters(&ncl, k_cluster, &cfg) == cudaSuccess && ncl >= 1) { csize = cs; break; }
                (void)cudaGetLastError();
            }
        }
        (void)cudaGetLastError();
        bool any = false;
        if (csize) {
            for (uint32_t i = c->first_pair_layer(); i < c->d; i++) {
                size_t need = dyn;
                if (plan_cluster_layer(c, i, csize, hc[i], need) && fixed + need <= F_SMEM_MAX) { dyn = need; fh.group[i] = 8; any = true; }
                else hc[i] = ClLayer{};
            }
        }
        if (any) {
            if (cudaMalloc(&fh.d_cl, hc.size() * sizeof(ClLayer)) != cudaSuccess) return VC_ERR_NOMEM;
            if (cudaMemcpy(fh.d_cl, hc.data(), hc.size() * sizeof(ClLayer), cudaMemcpyHostToDevice) != cudaSuccess) return VC_ERR_CUDA;
            fh.csize = csize; fh.cl_smem = fixed + dyn;
        }
    }
    if (cudaMemset(fh.d_stamps, 0, (size_t)(c->d + 1 + F_TRACE_WORDS) * 8) != cudaSuccess) return VC_ERR_CUDA;
    if (cudaMemcpy(fh.d_plan, h.data(), h.size() * sizeof(LayerPlan), cudaMemcpyHostToDevice) != cudaSuccess) return VC_ERR_CUDA;
    if (!all_cta.empty() &&
        cudaMemcpy(fh.d_cta, all_cta.data(), all_cta.size() * sizeof(CtaPlan), cudaMemcpyHostToDevice) != cudaSuccess) return VC_ERR_CUDA;
    if (cudaMemset(fh.d_slots, 0, (size_t)F_RING * F_SLOT_WORDS * 8) != cudaSuccess) return VC_ERR_CUDA;
    return VC_OK;
}

void fused_free(const vc_circuit *c) {
    std::lock_guard<std::mutex> lk(g_registry_mutex);
    for (size_t i = 0; i < g_fused.size(); i++)
        if (g_fused[i].first == c) {
            release(g_fused[i].second);
            g_fused.erase(g_fused.begin() + i);
            return;
        }
}

int fused_supported(const vc_circuit *c, uint32_t) { return find(c) != nullptr; }

// proves layers [begin, end) in ONE cooperative launch
int enqueue_layers_fused(vc_circuit *c, uint32_t begin, uint32_t end, uint64_t seed, uint64_t *d_tr, cudaStream_t st) {
    FusedHost *fh = find(c);
    if (!fh || begin < c->first_pair_layer()) return VC_ERR_STATE;
    // runs of layers by kernel group: {narrow, thin} -> k_fused<3>, {wide} -> k_fused<4>; more than F_MAX_RUNS runs -> one k_fused<7>
    std::vector<std::pair<uint32_t, int>> runs;          // (first layer, mask)
    for (uint32_t i = begin; i < end; i++) {
        const int m = fh->group[i];
        if (runs.empty() || runs.back().second != m || (m == 8 && i - runs.back().first >= CL_MAX_LAYERS)) runs.emplace_back(i, m);
    }
    if (runs.size() > F_MAX_RUNS || fh->single_kernel) {   // the all-kinds kernel cannot hold cluster layers: they keep their own launches
        bool has_cl = false;
        for (auto &r : runs) has_cl = has_cl || r.second == 8;
        if (!has_cl) { runs.clear(); runs.emplace_back(begin, 7); }
        else for (auto &r : runs) if (r.second != 8) r.second = 7;
    }
    if (begin == c->first_pair_layer()) {   // a proof starts: the rendezvous slots and their epoch start clean whatever an earlier, aborted launch left behind
        if (cudaMemsetAsync(fh->d_slots, 0, (size_t)F_RING * F_SLOT_WORDS * 8, st) != cudaSuccess ||
            cudaMemsetAsync(&c->d_state->bar_gen, 0, sizeof(unsigned int), st) != cudaSuccess) { (void)cudaGetLastError(); return VC_ERR_CUDA; }
    }
    uint64_t off = 0;
    for (size_t r = 0; r < runs.size(); r++) {
        const uint32_t b0 = runs[r].first, e0 = r + 1 < runs.size() ? runs[r + 1].first : end;
        FusedArgs a;
        a.L = fh->d_plan; a.d = c->d; a.begin = b0; a.end = e0; a.seed = seed; a.st = c->d_state; a.tr = d_tr + off;
        a.P = c->d_P; a.C = fh->d_C; a.T0 = c->d_T0; a.T1 = c->d_T1; a.Tg = fh->d_Tg; a.slots = fh->d_slots; a.stamps = fh->d_stamps;
        void *params[] = {&a};
        const int mask = runs[r].second;
        const void *fn = mask == 1 ? (const void *)k_fused<1> : mask == 2 ? (const void *)k_fused<2> : (mask == 4 ? (const void *)k_fused<4> : (const void *)k_fused<7>);
        cudaEvent_t ea = nullptr, eb = nullptr;
        if (g_profile) { cudaEventCreate(&ea); cudaEventCreate(&eb); cudaEventRecord(ea, st); }
        cudaError_t e;
        if (mask == 8) {
            ClArgs ca;
            ca.L = fh->d_plan; ca.cl = fh->d_cl; ca.d = c->d; ca.begin = b0; ca.end = e0; ca.csize = (uint32_t)fh->csize; ca.seed = seed;
            ca.st = c->d_state; ca.tr = d_tr + off; ca.stamps = fh->d_stamps;
            e = launch_cluster(ca, fh->csize, fh->cl_smem, st);
        } else {
            e = cudaLaunchCooperativeKernel(fn, dim3(fh->grid), dim3(FT), params, fh->smem, st);
        }
        if (g_profile) {
            cudaEventRecord(eb, st);
            prof_push(mask == 8 ? VC_K_CLUSTER : mask == 1 ? VC_K_FUSED_NARROW : mask == 2 ? VC_K_FUSED_THIN : VC_K_FUSED_WIDE, ea, eb);
        }
        g_launches.fetch_add(1, std::memory_order_relaxed);
        if (e != cudaSuccess) { (void)cudaGetLastError(); return VC_ERR_CUDA; }
        for (uint32_t i = b0; i < e0; i++) off += c->layer_words(i);
    }
    return VC_OK;
}

int fused_layer_kinds(const vc_circuit *c, uint32_t *h_kind) {
    FusedHost *fh = find(c);
    if (!fh) return VC_ERR_STATE;
    for (uint32_t i = 0; i < c->d; i++) {
        const int g = fh->group[i];
        h_kind[i] = g == 0 ? VC_K_ROUND : g == 8 ? VC_K_CLUSTER : g == 1 ? VC_K_FUSED_NARROW : g == 2 ? VC_K_FUSED_THIN : VC_K_FUSED_WIDE;
    }
    return VC_OK;
}

int fused_stamps(const vc_circuit *c, uint64_t *h, cudaStream_t st) {
    FusedHost *fh = find(c);
    if (!fh) return VC_ERR_STATE;
    if (cudaStreamSynchronize(st) != cudaSuccess) return VC_ERR_CUDA;
    return cudaMemcpy(h, fh->d_stamps, (size_t)(c->d + 1) * 8, cudaMemcpyDeviceToHost) == cudaSuccess ? VC_OK : VC_ERR_CUDA;
}

// a1 in one cooperative launch; returns VC_ERR_STATE when this circuit must use the per-layer kernels instead
int enqueue_eval_fused(vc_circuit *c, const uint64_t *d_input, uint64_t *d_outputs, cudaStream_t st) {
    FusedHost *fh = find(c);
    if (!fh || !fh->eval_ok) return VC_ERR_STATE;
    const LayerPlan *L = fh->d_plan; uint32_t d = c->d; DevState *S = c->d_state;
    int top = (int)c->first_pair_layer(), loc_top = fh->eval_loc_top;
    uint32_t loc_bl = fh->eval_loc_bl;
    void *params[] = {&L, &d, &d_input, &d_outputs, &S, &top, &loc_bl, &loc_top};
    cudaEvent_t ea = nullptr, eb = nullptr;
    if (g_profile) { cudaEventCreate(&ea); cudaEventCreate(&eb); cudaEventRecord(ea, st); }
    cudaError_t e = cudaLaunchCooperativeKernel((const void *)k_eval_all, dim3(fh->grid), dim3(EVAL_T), params, EVAL_SMEM, st);
    if (g_profile) { cudaEventRecord(eb, st); prof_push(VC_K_EVAL, ea, eb); }
    g_launches.fetch_add(1, std::memory_order_relaxed);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return VC_ERR_CUDA; }
    return VC_OK;
}

int fused_trace(const vc_circuit *c, uint64_t *h, uint32_t n_words, cudaStream_t st) {
    FusedHost *fh = find(c);
    if (!fh || n_words > F_TRACE_WORDS) return VC_ERR_ARG;
    if (cudaStreamSynchronize(st) != cudaSuccess) return VC_ERR_CUDA;
    return cudaMemcpy(h, fh->d_stamps + c->d + 1, (size_t)n_words * 8, cudaMemcpyDeviceToHost) == cudaSuccess ? VC_OK : VC_ERR_CUDA;
}

int enqueue_layer_fused(vc_circuit *c, uint32_t layer, uint64_t seed, uint64_t *d_tr, cudaStream_t st) {
    return enqueue_layers_fused(c, layer, layer + 1, seed, d_tr, st);
}

}  // namespace vc
