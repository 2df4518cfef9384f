// The generic instantiation of the fused pass (any code the handle accepts): pass_kernel.cuh.
#include "pass_kernel.cuh"

namespace qc {
void launch_pass_generic(const PassLaunch& L) { launch_pass_any(L); }
}  // namespace qc
