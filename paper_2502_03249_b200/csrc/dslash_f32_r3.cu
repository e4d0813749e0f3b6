// dslash_kernel instantiations: float, full 18-real links.
#include "dslash_inst.cuh"

namespace qcd {
cudaError_t launch_dslash_f32_r3(const DslashLaunch &d) { return launch_dslash_impl<float, 3>(d); }
} // namespace qcd
