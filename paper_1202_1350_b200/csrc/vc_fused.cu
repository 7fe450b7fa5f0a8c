// vc_fused.cu — on-chip ("fused") schedule of one GKR layer.  Placeholder until the persistent kernels land:
// reports "not supported" so every layer takes the streaming schedule.
#include "vc_circuit.hpp"

namespace vc {
int fused_init(vc_circuit *) { return VC_OK; }
int fused_supported(const vc_circuit *, uint32_t) { return 0; }
int enqueue_layer_fused(vc_circuit *, uint32_t, uint64_t, uint64_t *, cudaStream_t) { return VC_ERR_STATE; }
}  // namespace vc
