// tcgen05 assignment kernel (bf16, d = 128) -- placeholder until the TMA/tcgen05 contraction lands.
#include "common.cuh"
namespace pkv {
bool tc_assign_supported(const Dims&, const Hyper&) { return false; }
int launch_score_tc(const Dims& D, const Hyper& H, const Dev& V, const FrameArgs& F, cudaStream_t s) {
  return launch_score_simt(D, H, V, F, s);
}
}  // namespace pkv
