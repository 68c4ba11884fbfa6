// vegas_rtc.cu -- run-time compilation of a user integrand into the iterate / parity-hook kernels (NVRTC).
// the user hands a function of the points to `compile(integrand)`; here the function is C source
// compiled for sm_100a into the same kernel templates as the built-in integrands (csrc/vegas_user.cuh adapts it).
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include <cuda_runtime.h>
#include <dlfcn.h>
#include <nvrtc.h>

#include "../../include/vegas_b200.h"
#include "vegas_rtc.h"

namespace {

// directory of the library's kernel headers: csrc/ next to libvegas_b200.so
std::string csrc_dir()
{
    Dl_info info;
    if (!dladdr(reinterpret_cast<void*>(&vegas_create_custom), &info) || !info.dli_fname) return "";
    std::string p(info.dli_fname);
    const size_t k = p.find_last_of('/');
    return (k == std::string::npos ? std::string(".") : p.substr(0, k)) + "/csrc";
}

}  // namespace

int vegas_rtc_compile(int dim, int precision, const char* source, vegas_rtc_result* r, std::string* log)
{
    r->library = nullptr; r->iterate = nullptr; r->debug = nullptr;
    const std::string dir = csrc_dir();
    if (dir.empty()) { *log = "cannot locate the library's csrc/ directory (dladdr failed)"; return VEGAS_ECUDA; }
    // user code comes last: the kernel templates only need the prototype vegas_user.cuh declares
    std::string tu = "#define VEGAS_INTEGRAND __device__\n#define VEGAS_USER_DIM " + std::to_string(dim) + "\n";
    if (precision == VEGAS_FP64_U32) tu += "#define VEGAS_USER_U32 1\n";
    tu += "#include \"vegas_user.cuh\"\n#line 1 \"user_integrand\"\n";
    tu += source;
    tu += "\n";
    const std::string k_iter = "vegas::iterate_kernel<vegas::UserF, " + std::to_string(dim) + ", 0, -1, 1, 0, 1024, 1>";
    const std::string k_dbg = "vegas::debug_events_kernel<vegas::UserF, " + std::to_string(dim) + ">";

    nvrtcProgram prog;
    if (nvrtcCreateProgram(&prog, tu.c_str(), "vegas_user.cu", 0, nullptr, nullptr) != NVRTC_SUCCESS) { *log = "nvrtcCreateProgram failed"; return VEGAS_ECUDA; }
    nvrtcAddNameExpression(prog, k_iter.c_str());
    nvrtcAddNameExpression(prog, k_dbg.c_str());
    const std::string inc = "-I" + dir;
    const char* opts[] = {"--gpu-architecture=sm_100a", "-std=c++17", "--fmad=false", "-lineinfo", inc.c_str()};
    const nvrtcResult cr = nvrtcCompileProgram(prog, 5, opts);
    size_t ls = 0;
    nvrtcGetProgramLogSize(prog, &ls);
    if (ls > 1) { log->resize(ls); nvrtcGetProgramLog(prog, &(*log)[0]); }
    if (cr != NVRTC_SUCCESS) { nvrtcDestroyProgram(&prog); return VEGAS_EUNSUPPORTED; }
    const char *n_iter = nullptr, *n_dbg = nullptr;
    size_t cs = 0;
    if (nvrtcGetLoweredName(prog, k_iter.c_str(), &n_iter) != NVRTC_SUCCESS || nvrtcGetLoweredName(prog, k_dbg.c_str(), &n_dbg) != NVRTC_SUCCESS ||
        nvrtcGetCUBINSize(prog, &cs) != NVRTC_SUCCESS || cs == 0) {
        nvrtcDestroyProgram(&prog);
        *log += "\n(no cubin / kernel names from NVRTC)";
        return VEGAS_ECUDA;
    }
    std::vector<char> cubin(cs);
    nvrtcGetCUBIN(prog, cubin.data());
    cudaLibrary_t lib = nullptr;
    cudaKernel_t ki = nullptr, kd = nullptr;
    cudaError_t e = cudaLibraryLoadData(&lib, cubin.data(), nullptr, nullptr, 0, nullptr, nullptr, 0);
    if (e == cudaSuccess) e = cudaLibraryGetKernel(&ki, lib, n_iter);
    if (e == cudaSuccess) e = cudaLibraryGetKernel(&kd, lib, n_dbg);
    nvrtcDestroyProgram(&prog);
    if (e != cudaSuccess) {
        if (lib) cudaLibraryUnload(lib);
        *log += std::string("\nloading the compiled kernels failed: ") + cudaGetErrorString(e);
        (void)cudaGetLastError();
        return VEGAS_ECUDA;
    }
    r->library = lib; r->iterate = ki; r->debug = kd;
    return VEGAS_OK;
}
