// vc_fused.cu — kernel + host driver of the on-chip schedule (see vc_fused.cuh).
#include <algorithm>
#include <vector>

#include "vc_circuit.hpp"
#include "vc_fused_small.cuh"
#include "vc_fused_wide.cuh"

namespace vc {

__device__ __forceinline__ bool is_small(const FusedArgs &a, uint32_t layer) {
    return a.L[layer].log_n <= F_SMALL_N_LOG && a.L[layer + 1].log_n <= F_SMALL_T_LOG;
}

__global__ void __launch_bounds__(FT, 1) k_fused(FusedArgs a) {
    extern __shared__ __align__(16) uint8_t smem[];
    FusedCtx &cx = *reinterpret_cast<FusedCtx *>(smem);
    uint8_t *dyn = smem + sizeof(FusedCtx);
    const uint32_t tid = threadIdx.x;
    // ---- load (or start) the proof state
    if (a.begin == 0) {
        const uint32_t s0 = a.L[0].log_n;
        if (tid < s0) cx.z[tid] = fp61::draw(a.seed, tid);      // a2: z_0
        if (tid == 0) { cx.seed = a.seed; cx.ctr = s0; cx.claim = 0; }
    } else {
        if (tid < MAX_VARS) cx.z[tid] = a.st->z[tid];
        if (tid == 0) { cx.seed = a.seed; cx.ctr = a.st->ctr; cx.claim = a.st->claim; }
    }
    if (tid == 0) { cx.epoch = a.st->bar_gen; cx.v1 = 0; cx.v2 = 0; }
    __syncthreads();
    uint64_t *tr = a.tr;
    bool handoff = false;                         // CTA 0 ran narrow layers alone: publish its state first
    for (uint32_t layer = a.begin; layer < a.end; layer++) {
        const uint32_t s = a.L[layer + 1].log_n;
        if (blockIdx.x == 0 && tid == 0) a.stamps[layer] = globaltimer_ns();
        if (is_small(a, layer)) {
            if (blockIdx.x == 0) small_layer(a, cx, dyn, layer, tr);
            handoff = true;
        } else {
            if (handoff) {
                if (blockIdx.x == 0) {
                    if (tid < MAX_VARS) a.st->z[tid] = cx.z[tid];
                    if (tid == 0) { a.st->ctr = cx.ctr; a.st->claim = cx.claim; }
                }
                grid_allreduce(cx, a, 0);
                if (blockIdx.x != 0) {
                    if (tid < MAX_VARS) cx.z[tid] = __ldcg(&a.st->z[tid]);
                    if (tid == 0) { cx.ctr = __ldcg(&a.st->ctr); cx.claim = __ldcg(&a.st->claim); }
                }
                __syncthreads();
                handoff = false;
            }
            const uint32_t nch0 = (1u << a.L[layer].log_n) >> F_CHUNK_LOG, nch = nch0 ? nch0 : 1u;
            if ((nch + gridDim.x - 1) / gridDim.x <= (uint32_t)F_MAXK) wide_layer<true>(a, cx, dyn, layer, tr);
            else wide_layer<false>(a, cx, dyn, layer, tr);
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

struct FusedHost {
    LayerDesc *d_desc = nullptr;
    unsigned long long *d_slots = nullptr;
    uint64_t *d_stamps = nullptr;
    int grid = 0;
};
static std::vector<std::pair<const vc_circuit *, FusedHost>> g_fused;

static FusedHost *find(const vc_circuit *c) {
    for (auto &p : g_fused) if (p.first == c) return &p.second;
    return nullptr;
}

int fused_init(vc_circuit *c) {
    if (!c->coop_ok) return VC_OK;
    FusedHost fh;
    if (cudaFuncSetAttribute(k_fused, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)F_SMEM_BYTES) != cudaSuccess) {
        (void)cudaGetLastError();
        return VC_OK;                                // no fused schedule on this device; streaming still works
    }
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_fused, FT, F_SMEM_BYTES) != cudaSuccess || per_sm < 1) {
        (void)cudaGetLastError();
        return VC_OK;
    }
    fh.grid = c->sm_count;
    std::vector<LayerDesc> h(c->d + 1);
    for (uint32_t i = 0; i <= c->d; i++) {
        h[i].type = i < c->d ? c->d_type[i] : nullptr;
        h[i].in1 = i < c->d ? c->d_in1[i] : nullptr;
        h[i].in2 = i < c->d ? c->d_in2[i] : nullptr;
        h[i].V = c->d_V[i];
        h[i].log_n = c->logs[i];
        h[i].pad = 0;
    }
    if (cudaMalloc(&fh.d_desc, h.size() * sizeof(LayerDesc)) != cudaSuccess) return VC_ERR_NOMEM;
    if (cudaMalloc(&fh.d_slots, (size_t)F_RING * F_SLOT_WORDS * 8) != cudaSuccess) return VC_ERR_NOMEM;
    if (cudaMalloc(&fh.d_stamps, (size_t)(c->d + 1) * 8) != cudaSuccess) return VC_ERR_NOMEM;
    if (cudaMemset(fh.d_stamps, 0, (size_t)(c->d + 1) * 8) != cudaSuccess) return VC_ERR_CUDA;
    if (cudaMemcpy(fh.d_desc, h.data(), h.size() * sizeof(LayerDesc), cudaMemcpyHostToDevice) != cudaSuccess) return VC_ERR_CUDA;
    if (cudaMemset(fh.d_slots, 0, (size_t)F_RING * F_SLOT_WORDS * 8) != cudaSuccess) return VC_ERR_CUDA;
    g_fused.emplace_back(c, fh);
    return VC_OK;
}

void fused_free(const vc_circuit *c) {
    for (size_t i = 0; i < g_fused.size(); i++)
        if (g_fused[i].first == c) {
            cudaFree(g_fused[i].second.d_desc);
            cudaFree(g_fused[i].second.d_slots);
            cudaFree(g_fused[i].second.d_stamps);
            g_fused.erase(g_fused.begin() + i);
            return;
        }
}

int fused_supported(const vc_circuit *c, uint32_t) { return find(c) != nullptr; }

// proves layers [begin, end) in ONE cooperative launch
int enqueue_layers_fused(vc_circuit *c, uint32_t begin, uint32_t end, uint64_t seed, uint64_t *d_tr, cudaStream_t st) {
    FusedHost *fh = find(c);
    if (!fh) return VC_ERR_STATE;
    FusedArgs a;
    a.L = fh->d_desc; a.d = c->d; a.begin = begin; a.end = end; a.seed = seed; a.st = c->d_state; a.tr = d_tr;
    a.P = c->d_P; a.T0 = c->d_T0; a.T1 = c->d_T1; a.slots = fh->d_slots; a.stamps = fh->d_stamps;
    void *params[] = {&a};
    cudaEvent_t ea = nullptr, eb = nullptr;
    if (g_profile) { cudaEventCreate(&ea); cudaEventCreate(&eb); cudaEventRecord(ea, st); }
    cudaError_t e = cudaLaunchCooperativeKernel((const void *)k_fused, dim3(fh->grid), dim3(FT), params, F_SMEM_BYTES, st);
    if (g_profile) { cudaEventRecord(eb, st); prof_push(VC_K_FUSED_WIDE, ea, eb); }
    g_launches.fetch_add(1, std::memory_order_relaxed);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return VC_ERR_CUDA; }
    return VC_OK;
}

int fused_stamps(const vc_circuit *c, uint64_t *h, cudaStream_t st) {
    FusedHost *fh = find(c);
    if (!fh) return VC_ERR_STATE;
    if (cudaStreamSynchronize(st) != cudaSuccess) return VC_ERR_CUDA;
    return cudaMemcpy(h, fh->d_stamps, (size_t)(c->d + 1) * 8, cudaMemcpyDeviceToHost) == cudaSuccess ? VC_OK : VC_ERR_CUDA;
}

int enqueue_layer_fused(vc_circuit *c, uint32_t layer, uint64_t seed, uint64_t *d_tr, cudaStream_t st) {
    return enqueue_layers_fused(c, layer, layer + 1, seed, d_tr, st);
}

}  // namespace vc
