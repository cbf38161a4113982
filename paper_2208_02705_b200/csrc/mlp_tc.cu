// r360 -- grouped tiny-MLP on the tensor cores (tcgen05, bf16 operands, fp32 accumulate).
// PLACEHOLDER until the kernel lands: the library refuses precision mode 1.
#include "kernels.h"

namespace r360 {

size_t tc_pack_stride(const NetShape&) { return 0; }
void tc_pack_subfield(const NetShape&, const float*, void*) {}

cudaError_t launch_mlp_tc(const GridParams&, const FrameParams&, const ChunkBuffers&, const NetShape&,
                          const void*, size_t, const SubfieldFrame*, int, int, int, cudaStream_t) {
  return cudaErrorNotSupported;
}

}  // namespace r360
