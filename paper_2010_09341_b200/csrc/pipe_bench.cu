// pipe_bench.cu -- vegas_pipe_rate(): instruction-throughput microbenchmarks of the SM pipes the Vegas hot
// path runs on.  They are the measured denominators of the roofline bench.py reports:
// the path moves no HBM bytes per event and is no tensor-core contraction, so its bound is the issue rate of
// the FP64 pipe (DFMA/DADD/DMUL), of the FP32 pipes (FFMA), of the wide integer multiplier Philox needs
// (IMAD.WIDE.U32), of the logic pipe (LOP3) and of the shared-memory compare-and-swap an fp64 histogram
// update is on sm_100a.  Measured in the same process, right before the timed region, because the SM clock
// under load is not the nominal one.
#include <cstdint>
#include <cuda_runtime.h>

#include "../../include/vegas_b200.h"

namespace {

constexpr int kChains = 8;    // independent dependency chains per thread
constexpr int kUnroll = 16;   // operations per chain per loop trip

template <int KIND>
__global__ void __launch_bounds__(1024, 1) pipe_kernel(int iters, unsigned long long* out, uint32_t seed)
{
    extern __shared__ double sh[];                     // KIND 4, 6, 7: [32 cells][32 lanes]; KIND 5: [2000 cells][8 replicas]
    const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    double d[kChains], e3[kChains], g3[kChains];
    float f[kChains];
    unsigned long long w[kChains];
    uint32_t u[kChains], v[kChains];
#pragma unroll
    for (int c = 0; c < kChains; ++c) {
        d[c] = 1.0 + 1e-9 * (t + c);
        e3[c] = 1.0 + 1e-12 * (t + 3 * c);              // KIND 8: per-thread register operands
        g3[c] = 1e-9 * (t + c + 1);
        f[c] = 1.0f + 1e-6f * (t + c);
        w[c] = static_cast<unsigned long long>(t * 7u + c) * 0x9E3779B97F4A7C15ull + seed;
        u[c] = t * 31u + c + seed;
        v[c] = t * 17u + c * 3u + seed;
    }
    if (KIND >= 4) {
        const int words = (KIND == 5) ? 2000 * 8 : 32 * 32;
        for (int i = threadIdx.x; i < words; i += blockDim.x) sh[i] = 0.0;
        __syncthreads();
    }
    const double da = 1.0000001, db = 1e-9;
    const float fa = 1.0001f, fb = 1e-6f;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int j = 0; j < kUnroll; ++j) {
#pragma unroll
            for (int c = 0; c < kChains; ++c) {
                if (KIND == 0) d[c] = __fma_rn(d[c], da, db);
                if (KIND == 1) f[c] = __fmaf_rn(f[c], fa, fb);
                if (KIND == 2) asm volatile("mad.wide.u32 %0, %1, %2, 0;" : "=l"(w[c]) : "r"(static_cast<uint32_t>(w[c] >> 32)), "r"(0xD2511F53u));
                if (KIND == 3) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(u[c]) : "r"(v[c]), "r"(seed));
                if (KIND == 4) {
                    // one fp64 histogram update: lane-indexed replica (conflict-free within the warp), pseudo-random cell
                    u[c] = u[c] * 1664525u + 1013904223u;
                    atomicAdd(&sh[((u[c] >> 27) << 5) + (threadIdx.x & 31)], db);
                }
                if (KIND == 5) {
                    // the same with the layout configs[3] is forced into (2000 cells, R = 8: four lanes of a warp share a
                    // replica and collide when they draw the same cell of 100 -- here one of 100 consecutive cells)
                    u[c] = u[c] * 1664525u + 1013904223u;
                    atomicAdd(&sh[(((u[c] >> 16) % 100u + 100u * c) << 3) + (threadIdx.x & 7)], db);
                }
                if (KIND == 6) {
                    // what the update would cost WITHOUT atomicity (a word that only this lane of this warp may touch:
                    // not available to the kernel -- it would take 32 replicas per warp): LDS.64, DADD, STS.64
                    u[c] = u[c] * 1664525u + 1013904223u;
                    double* p = &sh[((u[c] >> 27) << 5) + (threadIdx.x & 31)];
                    asm volatile("{\n\t.reg .f64 t;\n\tld.volatile.f64 t, [%0];\n\tadd.rn.f64 t, t, %1;\n\tst.volatile.f64 [%0], t;\n\t}" :: "l"(p), "d"(db) : "memory");
                }
                if (KIND == 8)      // DFMA with three distinct register operands (a Horner step whose coefficient is in a register)
                    asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(d[c]) : "d"(e3[c]), "d"(g3[c]));
                if (KIND == 9) {   // the event loop's ratio: 3 (IMAD.WIDE + LOP3) Philox half-rounds, 2 IMAD, 5 fp64, 5 LOP3
                    if (c < 3) {
                        const uint32_t x = static_cast<uint32_t>(w[c] >> 32) ^ static_cast<uint32_t>(w[c]) ^ seed;
                        asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(w[c]) : "r"(x), "r"(0xD2511F53u));
                    }
                    if (c >= 3 && c < 5) asm volatile("mad.lo.u32 %0, %0, %1, %1;" : "+r"(u[c]) : "r"(seed));
                    if (c < 5) asm volatile("fma.rn.f64 %0, %0, %1, %1;" : "+d"(d[c]) : "d"(e3[c]));
                    // logic operations chained across the chains (u[c] with its neighbour), so that none can be merged
                    if (c >= 3) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(u[c]) : "r"(u[c == 7 ? 3 : c + 1]), "r"(seed));
                }
                if (KIND == 7) {
                    // the native shared-memory atomic: 32-bit integer add (cannot hold the histogram's dynamic range)
                    u[c] = u[c] * 1664525u + 1013904223u;
                    atomicAdd(reinterpret_cast<unsigned int*>(sh) + ((u[c] >> 27) << 5) + (threadIdx.x & 31), u[c] >> 20);
                }
            }
        }
    }
    unsigned long long acc = 0;
#pragma unroll
    for (int c = 0; c < kChains; ++c)
        acc += static_cast<unsigned long long>(__double_as_longlong(d[c])) + __float_as_uint(f[c]) + w[c] + u[c] + v[c] +
               static_cast<unsigned long long>(__double_as_longlong(e3[c])) + static_cast<unsigned long long>(__double_as_longlong(g3[c]));
    if (acc == 0x1234567ull) out[t] = acc;             // never true in practice: keeps the chains alive
}

template <int KIND>
cudaError_t time_kind(int sms, int iters, unsigned long long* out, cudaStream_t st, double* rate)
{
    const int blocks = sms * 2, threads = 1024;
    const size_t smem = (KIND == 5) ? 2000 * 8 * sizeof(double) : (KIND >= 4) ? 32 * 32 * sizeof(double) : 0;
    if (KIND == 5) cudaFuncSetAttribute(pipe_kernel<KIND>, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
    cudaEvent_t e0, e1;
    cudaError_t e = cudaEventCreate(&e0);
    if (e != cudaSuccess) return e;
    e = cudaEventCreate(&e1);
    if (e != cudaSuccess) { cudaEventDestroy(e0); return e; }
    float best = 0.f;
    for (int r = 0; r < 3 && e == cudaSuccess; ++r) {  // first pass warms up; best of the next two
        cudaEventRecord(e0, st);
        pipe_kernel<KIND><<<blocks, threads, smem, st>>>(iters, out, 12345u + r);
        cudaEventRecord(e1, st);
        e = cudaEventSynchronize(e1);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        if (r > 0 && (best == 0.f || ms < best)) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (e != cudaSuccess) return e;
    // instructions per pass over the chains: one per chain, except the mixed group of KIND 9 (18)
    const double per_pass = (KIND == 9) ? 18.0 : static_cast<double>(kChains);
    const double ops = static_cast<double>(iters) * kUnroll * per_pass * blocks * threads;
    *rate = ops / (best * 1e-3);
    return cudaSuccess;
}

}  // namespace

extern "C" int vegas_pipe_rate(int pipe, void* cuda_stream, double* thread_instr_per_s)
{
    if (!thread_instr_per_s) return VEGAS_EINVAL;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) {
        (void)cudaGetLastError();
        return VEGAS_ECUDA;
    }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    unsigned long long* out = nullptr;
    if (cudaMalloc(reinterpret_cast<void**>(&out), static_cast<size_t>(sms) * 2 * 1024 * 8) != cudaSuccess) return VEGAS_ECUDA;
    cudaError_t e = cudaErrorInvalidValue;
    switch (pipe) {
        case VEGAS_PIPE_DFMA: e = time_kind<0>(sms, 1000, out, st, thread_instr_per_s); break;
        case VEGAS_PIPE_FFMA: e = time_kind<1>(sms, 2000, out, st, thread_instr_per_s); break;
        case VEGAS_PIPE_IMAD_WIDE: e = time_kind<2>(sms, 500, out, st, thread_instr_per_s); break;
        case VEGAS_PIPE_LOP3: e = time_kind<3>(sms, 1000, out, st, thread_instr_per_s); break;
        case VEGAS_PIPE_SHARED_F64_ADD: e = time_kind<4>(sms, 100, out, st, thread_instr_per_s); break;
        case VEGAS_PIPE_SHARED_F64_ADD_R8: e = time_kind<5>(sms, 50, out, st, thread_instr_per_s); break;
        case VEGAS_PIPE_SHARED_F64_RMW_PLAIN: e = time_kind<6>(sms, 100, out, st, thread_instr_per_s); break;
        case VEGAS_PIPE_SHARED_U32_ADD: e = time_kind<7>(sms, 100, out, st, thread_instr_per_s); break;
        case VEGAS_PIPE_DFMA_3REG: e = time_kind<8>(sms, 500, out, st, thread_instr_per_s); break;
        case VEGAS_PIPE_MIX_EVENT_LOOP: e = time_kind<9>(sms, 500, out, st, thread_instr_per_s); break;
        default: cudaFree(out); return VEGAS_EINVAL;
    }
    cudaFree(out);
    return e == cudaSuccess ? VEGAS_OK : VEGAS_ECUDA;
}
