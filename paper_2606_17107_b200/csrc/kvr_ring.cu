// kvr_ring.cu -- TMA-ring kernel (placeholder until the first GPU parity run of the generic kernel).
#include "kvr_common.cuh"
namespace kvr {
bool ring_supported(const CallParams&, const SegDev*, const char** why) { if (why) *why = "not built yet"; return false; }
cudaError_t launch_ring(const CallParams&, const RingConfig&, int, cudaStream_t, int*, int*, int*) { return cudaErrorNotSupported; }
}  // namespace kvr
