// Runtime descriptor of one Dslash launch and the per-(precision, link rows) launchers.
// The kernel template (dslash.cuh) is instantiated in four translation units
// (dslash_f64_r3.cu, dslash_f64_r2.cu, dslash_f32_r3.cu, dslash_f32_r2.cu) so that they build
// in parallel; qcd_api.cu only fills this struct.
#pragma once
#include <cuda_runtime.h>

#include "lattice.cuh"
#include "reduce.cuh"

namespace qcd {

struct DslashLaunch {
    int mode;              // 0: D, 1: m^2 v - D, 2: mode 1 + Re<v,out> partials + alpha (dslash.cuh)
    int tg;                // 1: temporal-gauge links (time links with x3 != 0 are the identity, not read)
    int nrhs;              // 1 .. MAXRHS vectors sharing every link load
    int variant;           // block-shape knob for the nrhs = 1, tg = 0 kernels (bench sweeps)
    Lattice L;
    int parity;            // parity of the output sites
    const void *U;
    const void *in[MAXRHS];
    void *out[MAXRHS];
    const void *v[MAXRHS];
    double m2;
    double *partials;
    CgScalars *scal;
    int check_flag;
    cudaStream_t stream;
};

// Each returns cudaErrorInvalidValue for an unsupported (mode, nrhs) combination, else the
// launch error state.  NROW = 3: full 18-real links; NROW = 2: two-row links.
cudaError_t launch_dslash_f64_r3(const DslashLaunch &d);
cudaError_t launch_dslash_f64_r2(const DslashLaunch &d);
cudaError_t launch_dslash_f32_r3(const DslashLaunch &d);
cudaError_t launch_dslash_f32_r2(const DslashLaunch &d);

} // namespace qcd
