// TEST INFRASTRUCTURE ONLY -- symbols of translation units that are not part of the emulated build.
#include "include/cuda_runtime.h"
#include "../../paper_2308_10868_b200/csrc/nrr_internal.cuh"

namespace nrr {
int fp32_peak_measure(double *out_tflops, cudaStream_t)      // the FFMA microbenchmark measures hardware
{
    *out_tflops = 0.0;
    set_error("the FFMA microbenchmark does not exist in the emulated build");
    return NRR_E_CUDA;
}
int fp32_microbench(double out[7], cudaStream_t)
{
    for (int i = 0; i < 7; ++i) out[i] = 0.0;
    set_error("the FP32 microbenchmarks do not exist in the emulated build");
    return NRR_E_CUDA;
}
}  // namespace nrr
