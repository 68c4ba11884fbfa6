// vegas_user.cuh -- adapter of a user-supplied integrand to the streaming integrand interface of
// vegas_device.cuh.  Included only in the translation unit vegas_create_custom() hands to NVRTC (PAPER.md:L72-L78:
// the user writes `def integrand(xarr, **kwargs)` and calls `compile(integrand)`; here the user writes
//     VEGAS_INTEGRAND double vegas_user_integrand(const double* x, int dim, const double* params) { ... }
// in the subset of C that is also valid CUDA device code, and the library compiles it into the same iterate
// kernel template as the built-in integrands).  VEGAS_USER_DIM is defined on the NVRTC command line.
#pragma once
#include "vegas_kernels.cuh"

VEGAS_INTEGRAND double vegas_user_integrand(const double* x, int dim, const double* params);

namespace vegas {

struct UserIntegrand {
    using real = double;
    static constexpr int kId = 5;
    static constexpr bool kU32 = false;
    static constexpr bool kHasCut = false;
    double x[VEGAS_USER_DIM];
    __device__ __forceinline__ void begin(const IntegrandConsts&) {}
    __device__ __forceinline__ void coord(int k, double xv, const IntegrandConsts&) { x[k] = xv; }
    __device__ __forceinline__ bool precheck(const IntegrandConsts&) const { return true; }
    __device__ __forceinline__ double end(const IntegrandConsts& c, int d) const
    {
        return vegas_user_integrand(x, d, c.user_params);
    }
};

#ifdef VEGAS_USER_U32
using UserF = U32<UserIntegrand>;
#else
using UserF = UserIntegrand;
#endif

}  // namespace vegas
