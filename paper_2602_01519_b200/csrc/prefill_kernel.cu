// placeholder until the tcgen05 kernel lands
#include "kernels.h"
namespace comb {
bool prefill_supported(int, int, int) { return false; }
cudaError_t prefill_encode_kv_maps(const PoolGeom &, TensorMapBlob *, TensorMapBlob *) { return cudaErrorNotSupported; }
cudaError_t prefill_encode_q_map(const void *, int64_t, int, int, int, TensorMapBlob *) { return cudaErrorNotSupported; }
cudaError_t launch_prefill(const PoolGeom &, int, const LinkView &, const PrefillMaps &, const PrefillItem *, int, int,
                           float, void *, float *, cudaStream_t) { return cudaErrorNotSupported; }
}  // namespace comb
