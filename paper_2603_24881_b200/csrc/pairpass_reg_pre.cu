// Register form of the density pre-pass: see pairpass_reg_kernel.cuh.
#include "pairpass_reg_kernel.cuh"

namespace gpw {
cudaError_t launch_pair_reg_pre(const pp::PassArgs &A, cudaStream_t st) { return launch_pair_reg_t<false>(A, st); }
}  // namespace gpw
