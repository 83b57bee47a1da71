// Register form of the Fock post-pass: see pairpass_reg_kernel.cuh.
#include "pairpass_reg_kernel.cuh"

namespace gpw {
cudaError_t launch_pair_reg_post(const pp::PassArgs &A, cudaStream_t st) { return launch_pair_reg_t<true>(A, st); }
}  // namespace gpw
