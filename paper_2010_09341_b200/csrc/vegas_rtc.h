// vegas_rtc.h -- internal interface between vegas_api.cu and vegas_rtc.cu (not part of the C ABI).
#pragma once
#include <string>

#include <cuda_runtime.h>

struct vegas_rtc_result {
    cudaLibrary_t library;
    cudaKernel_t iterate;   // iterate_kernel<UserF, dim, 0, -1, 1, 0, 1024, 1>
    cudaKernel_t debug;     // debug_events_kernel<UserF, dim>
};

// Compiles `source` (see vegas_create_custom) with NVRTC for sm_100a and loads the kernels.  `log` receives the
// compiler output.  Returns VEGAS_OK, VEGAS_EUNSUPPORTED (compilation failed) or VEGAS_ECUDA.
int vegas_rtc_compile(int dim, int precision, const char* source, vegas_rtc_result* result, std::string* log);
