// dslash_kernel instantiations: double, two-row links.
#include "dslash_inst.cuh"

namespace qcd {
cudaError_t launch_dslash_f64_r2(const DslashLaunch &d) { return launch_dslash_impl<double, 2>(d); }
} // namespace qcd
