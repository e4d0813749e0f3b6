// dslash_kernel instantiations: double, full 18-real links.
#include "dslash_inst.cuh"

namespace qcd {
cudaError_t launch_dslash_f64_r3(const DslashLaunch &d) { return launch_dslash_impl<double, 3>(d); }
} // namespace qcd
