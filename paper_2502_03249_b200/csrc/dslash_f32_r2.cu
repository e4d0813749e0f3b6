// dslash_kernel instantiations: float, two-row links.
#include "dslash_inst.cuh"

namespace qcd {
cudaError_t launch_dslash_f32_r2(const DslashLaunch &d) { return launch_dslash_impl<float, 2>(d); }
} // namespace qcd
