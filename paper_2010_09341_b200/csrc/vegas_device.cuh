// vegas_device.cuh -- per-event device functions of the Vegas hot path (sm_100a).
//
// Steps S1-S4 of the reading in DESIGN.md / SURVEY.md 8.c (the paper only names the method,
// PAPER.md:L11, L21-L25, L88): S1 counter-based random stream, S2 integer-exact grid map, S3 integrand,
// S4 weight.  Everything here stays in registers; the only memory touched is the (lo, wd) mapping table
// in shared memory.  No code is shared with oracle/.
#pragma once
#ifdef __CUDACC_RTC__
// run-time compilation of a user integrand (vegas_create_custom, NVRTC): no host headers
typedef unsigned int uint32_t;
typedef int int32_t;
typedef unsigned long long uint64_t;
namespace std {
template <bool B, class T, class F> struct conditional { typedef T type; };
template <class T, class F> struct conditional<false, T, F> { typedef F type; };
}
#else
#include <cstdint>
#include <type_traits>
#include <cuda_runtime.h>
#endif

namespace vegas {

constexpr int kMaxDim = 32;

// ------------------------------------------------------------------------------------------------
// Kernel arguments (one struct, passed __grid_constant__ so that round keys and integrand constants
// are constant-bank operands).
// ------------------------------------------------------------------------------------------------
struct IntegrandConsts {
    // I0 / I1 (gauss_sym, gauss_double): C = (alpha sqrt(pi))^-d, a2 = 1/alpha^2, mu[2]
    double gC, ga2, gmu0, gmu1, ghalfC;
    // I3 (lo_2to2): s, L = log(tau), cos_cut, pdf_a, L^2/s
    double hs, hL, hcut, ha, hLLs;   // hLLs = L^2/s
    // I2 (genz_osc_peak), fp32: phi, c_k, w_k = 1/c_k^2
    float zphi;
    float zc[kMaxDim];
    float zw[kMaxDim];
    // user integrand compiled at run time (vegas_create_custom): its parameters
    double user_params[16];
    // lo_2to2_tab: the tabulated PDF (device pointer into the workspace, vegas_set_table) and its length
    const double* tab;
    int ntab;
    // exp_f64: log2(e), 1.5 * 2^52, -ln2 (high, low), 1/13! ... 1/2!  (kernel parameters, so that every use is a
    // uniform-register operand of the fused multiply-add and costs neither a register nor a move)
    double ec[16];
};

#ifndef __CUDACC_RTC__
// The table behind IntegrandConsts::ec, filled by the host (vegas_api.cu).
inline void fill_exp_consts(double* ec)
{
    ec[0] = 0x1.71547652b82fep+0;            // log2(e), rounded
    ec[1] = 0x1.8p52;                        // 1.5 * 2^52: adding it leaves round(x log2 e) in the low word
    ec[2] = -0x1.62e42fefa39efp-1;           // -rnd(ln 2)
    ec[3] = -0x1.abc9e3b39803fp-56;          // -rnd(ln 2 - rnd(ln 2))
    double f = 1.0;
    for (int n = 2; n <= 13; ++n) f *= static_cast<double>(n);      // 13! = 6227020800, exact
    for (int n = 13; n >= 2; --n) { ec[4 + (13 - n)] = 1.0 / f; f /= static_cast<double>(n); }   // 1/n!: one rounding each
}
#endif


constexpr int kMaxUserParams = 16;

struct IterArgs {
    const void* table;     // device: (lo, wd) per cell, [dim][nbins], double2 (fp64) or float2 (fp32)
    double* hist;          // device: H[dim][nbins], accumulated with global fp64 reductions at CTA exit
    double* slots;         // device: per-CTA compensated accumulators [grid][4] = S1.hi, S1.lo, S2.hi, S2.lo
    unsigned long long* npass;  // device: number of events whose integrand was not cut away
    uint32_t e_lo_first;   // low word of the first global event index of this launch
    uint32_t e_hi;         // high word (uniform within a launch: launches never straddle 2^32)
    uint32_t count;        // events in this launch (<= 2^31)
    uint32_t iteration;    // Philox counter word 2 (used when iter_ptr is NULL)
    const uint32_t* iter_ptr;  // device: the counter lives in memory (CUDA-graph replays of run_integration)
    // S6 runs in the CTA that finishes last over all launches of the iteration (ticket counter):
    unsigned int* ticket;      // device: CTAs finished so far (zeroed with the accumulators)
    unsigned int total_ctas;   // CTAs of all launches of this iteration
    double* slots0;            // base of the slot regions; fin_lanes regions of stride fin_stride, fin_used slots each
    int fin_lanes, fin_stride, fin_used;
    unsigned long long n_events;   // events of the whole iteration; 0: this launch is a shard (no S6, NEXT-2)
    double* partials;          // device: S1.hi, S1.lo, S2.hi, S2.lo, npass, pad[3] -- the 8-double header in front of H
    double* result;            // device: I, sigma, S1, S2, npass, n
    uint32_t* dev_iter;        // graph replays: advanced by S6 (NULL otherwise)
    double* ring;              // graph replays: (I, sigma) log (NULL otherwise)
    int ring_len;
    // fused step (vegas_step_enqueue): the CTA that finishes last also refines (S7) and leaves the accumulators clean
    double refine_alpha;       // < 0: no refinement in this kernel
    double* edges;             // device: master edges E[dim][nbins+1]
    double* new_edges;         // device: candidate edges
    int* status;               // device: refinement status words (rejected count, -, latest outcome)
    int precision;             // 0: fp64 table, 1: fp32 table
    int smem_bytes;            // dynamic shared memory of this launch (reused by the refinement)
    uint32_t rk0[10], rk1[10];  // Philox round keys: k + r * Weyl
    int dim, nbins;
    int rshift;            // log2 of the number R of lane-indexed histogram replicas in shared memory
    IntegrandConsts ic;
};

// ------------------------------------------------------------------------------------------------
// S1 -- Philox4x32-10 (Salmon et al. 2011): multipliers 0xD2511F53 / 0xCD9E8D57, ten rounds, round
// function (hi(M1 c2)^c1^k0, lo(M1 c2), hi(M0 c0)^c3^k1, lo(M0 c0)).  Round keys come precomputed.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void mulhilo(uint32_t a, uint32_t b, uint32_t& hi, uint32_t& lo)
{
    const uint64_t p = static_cast<uint64_t>(a) * static_cast<uint64_t>(b);      // one IMAD.WIDE.U32
    hi = static_cast<uint32_t>(p >> 32);
    lo = static_cast<uint32_t>(p);
}

__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              const IterArgs& a, uint32_t r[4])
{
#pragma unroll
    for (int i = 0; i < 10; ++i) {
        uint32_t h0, l0, h1, l1;
        mulhilo(0xD2511F53u, c0, h0, l0);
        mulhilo(0xCD9E8D57u, c2, h1, l1);
        const uint32_t n0 = h1 ^ c1 ^ a.rk0[i];
        const uint32_t n2 = h0 ^ c3 ^ a.rk1[i];
        c0 = n0; c1 = l1; c2 = n2; c3 = l0;
    }
    r[0] = c0; r[1] = c1; r[2] = c2; r[3] = c3;
}

// ------------------------------------------------------------------------------------------------
// S2 -- integer-exact bin rule and interpolation.
//   fp64: m = 52-bit mantissa from words (lo, hi); p = m*N exactly; i = p>>52; frac = (p mod 2^52)/2^52.
//         m*N = hi*(N<<20) + (lo>>12)*N   (N < 2^12, so every term fits 64 bits).
//   fp32: m = r>>9 (23 bits); p = m*N (N < 2^9); i = p>>23; frac = (p mod 2^23)/2^23.
// frac is built by OR-ing the remainder under the exponent of 1.0 and subtracting 1.0 (one exact add).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void bin_frac64(uint32_t w_lo, uint32_t w_hi, uint32_t N, int& i, double& frac)
{
    // (w_lo>>12)*N < 2^32: a 32-bit multiply, then one wide multiply-add
    const uint32_t lp = (w_lo >> 12) * N;
    uint32_t plo, phi;                                   // p = w_hi * (N << 20) + lp: wide multiply, add with carry
    asm("{\n\t.reg .u64 t;\n\t.reg .u32 tl, th;\n\tmul.wide.u32 t, %2, %3;\n\tmov.b64 {tl, th}, t;\n\t"
        "add.cc.u32 %0, tl, %4;\n\taddc.u32 %1, th, 0;\n\t}" : "=r"(plo), "=r"(phi) : "r"(w_hi), "r"(N << 20), "r"(lp));
    i = static_cast<int>(phi >> 20);
    // the bin sits in bits 20.. of phi: OR-ing it into the exponent field of 1.0 (0x3FF: ten low bits set) changes
    // nothing as long as the bin index has at most ten bits
    const uint32_t fh = (N <= 1024u) ? (phi | 0x3FF00000u) : ((phi & 0x000FFFFFu) | 0x3FF00000u);
    frac = __dadd_rn(__hiloint2double(static_cast<int>(fh), static_cast<int>(plo)), -1.0);
}

// 32-bit-uniform stream mode (VEGAS_FP64_U32): m = w (32 bits), p = m*N, i = p>>32, frac = (p mod 2^32)/2^32.
__device__ __forceinline__ void bin_frac64_u32(uint32_t w, uint32_t N, int& i, double& frac)
{
    const uint64_t p = static_cast<uint64_t>(w) * static_cast<uint64_t>(N);
    const uint32_t lo = static_cast<uint32_t>(p);
    i = static_cast<int>(p >> 32);
    frac = __dadd_rn(__hiloint2double(static_cast<int>(0x3FF00000u | (lo >> 12)), static_cast<int>(lo << 20)), -1.0);
}

__device__ __forceinline__ void bin_frac32(uint32_t w, uint32_t N, int& i, float& frac)
{
    const uint32_t p = (w >> 9) * N;
    i = static_cast<int>(p >> 23);
    frac = __fadd_rn(__uint_as_float((p & 0x007FFFFFu) | 0x3F800000u), -1.0f);
}

// ------------------------------------------------------------------------------------------------
// Shared memory by 32-bit shared-window address: one register per address, cell offsets known at compile time
// fold into the instruction's immediate, and nothing is spent on generic-to-shared conversion in the event loop.
// The mapping table is read-only while events are processed (plain asm: the compiler may schedule the loads).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_addr(const void* p) { return static_cast<uint32_t>(__cvta_generic_to_shared(p)); }

__device__ __forceinline__ void lds_cell(uint32_t addr, double& lo, double& wd)
{
    asm("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(lo), "=d"(wd) : "r"(addr));
}
__device__ __forceinline__ void lds_cell(uint32_t addr, float& lo, float& wd)
{
    asm("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(lo), "=f"(wd) : "r"(addr));
}
__device__ __forceinline__ void ldg_cell(const void* table, int cell, double& lo, double& wd)
{
    const double2 t = static_cast<const double2*>(table)[cell];
    lo = t.x; wd = t.y;
}
__device__ __forceinline__ void ldg_cell(const void* table, int cell, float& lo, float& wd)
{
    const float2 t = static_cast<const float2*>(table)[cell];
    lo = t.x; wd = t.y;
}

// ------------------------------------------------------------------------------------------------
// exp for the built-in fp64 integrands: k = round(x log2 e) by the 1.5 * 2^52 shift, r = x - k ln 2 in two fused
// steps (ln 2 split in a rounded part and its remainder), e^r by the degree-13 Taylor polynomial (|r| <= 0.347:
// remainder 6e-18 relative), scaled by 2^k through the exponent field.  Within about one unit in the last place of
// the correctly rounded value (the tests allow 2e-15 relative against the oracle's libm).  Every constant is a
// kernel parameter: on sm_100a a DFMA with three register operands takes three issue cycles, one with two registers
// and a uniform operand under two (measured), and CUDA's exp() rebuilds its thirteen constants
// in registers with two moves each.  Outside |x| < 700 (overflow, subnormal results) the library routine is used.
// ------------------------------------------------------------------------------------------------
template <int NX>
__device__ __forceinline__ void exp_f64(const double (&x)[NX], double (&y)[NX], const IntegrandConsts& c)
{
    bool in_range = true;
#pragma unroll
    for (int j = 0; j < NX; ++j) in_range = in_range && (fabs(x[j]) < 700.0);
    if (!in_range) {
#pragma unroll
        for (int j = 0; j < NX; ++j) y[j] = exp(x[j]);
        return;
    }
    // the NX evaluations run side by side: one load of each constant, NX independent chains
    int k[NX];
    double r[NX], p[NX];
#pragma unroll
    for (int j = 0; j < NX; ++j) {
        const double t = __fma_rn(x[j], c.ec[0], c.ec[1]);
        k[j] = __double2loint(t);
        const double kf = __dsub_rn(t, c.ec[1]);
        r[j] = __fma_rn(kf, c.ec[3], __fma_rn(kf, c.ec[2], x[j]));
        p[j] = c.ec[4];
    }
#pragma unroll
    for (int i = 5; i < 16; ++i)
#pragma unroll
        for (int j = 0; j < NX; ++j) p[j] = __fma_rn(p[j], r[j], c.ec[i]);
#pragma unroll
    for (int j = 0; j < NX; ++j) {
        p[j] = __fma_rn(p[j], r[j], 1.0);
        p[j] = __fma_rn(p[j], r[j], 1.0);
        y[j] = __hiloint2double(__double2hiint(p[j]) + (k[j] << 20), __double2loint(p[j]));
    }
}

// ------------------------------------------------------------------------------------------------
// S3 -- integrands as streaming accumulators: begin(), coord(k, x_k) in ascending k, end() -> f.
// Evaluation order is the normative one of SURVEY.md 8.c I0-I4; every fused multiply-add is explicit
// and every other product/sum uses the non-contracting intrinsics.
// ------------------------------------------------------------------------------------------------
struct GaussSym {            // I0, BASELINE.json configs[0]
    using real = double;
    static constexpr int kId = 0;
    static constexpr bool kU32 = false;
    static constexpr bool kHasCut = false;   // true: f = 0 for events the integrand's cuts reject
    double s;
    __device__ __forceinline__ void begin(const IntegrandConsts&) { s = 0.0; }
    __device__ __forceinline__ void coord(int, double x, const IntegrandConsts& c)
    {
        const double dx = __dsub_rn(x, c.gmu0);
        s = __fma_rn(dx, dx, s);
    }
    __device__ __forceinline__ bool precheck(const IntegrandConsts&) const { return true; }
    __device__ __forceinline__ double end(const IntegrandConsts& c, int) const
    {
        const double x[1] = {-__dmul_rn(s, c.ga2)};
        double e[1];
        exp_f64(x, e, c);
        return __dmul_rn(c.gC, e[0]);
    }
};

struct GaussDouble {         // I1, BASELINE.json configs[1], [2]
    using real = double;
    static constexpr int kId = 1;
    static constexpr bool kU32 = false;
    static constexpr bool kHasCut = false;   // true: f = 0 for events the integrand's cuts reject
    double s1, s2;
    __device__ __forceinline__ void begin(const IntegrandConsts&) { s1 = 0.0; s2 = 0.0; }
    __device__ __forceinline__ void coord(int, double x, const IntegrandConsts& c)
    {
        const double d1 = __dsub_rn(x, c.gmu0), d2 = __dsub_rn(x, c.gmu1);
        s1 = __fma_rn(d1, d1, s1);
        s2 = __fma_rn(d2, d2, s2);
    }
    __device__ __forceinline__ bool precheck(const IntegrandConsts&) const { return true; }
    __device__ __forceinline__ double end(const IntegrandConsts& c, int) const
    {
        const double x[2] = {-__dmul_rn(s1, c.ga2), -__dmul_rn(s2, c.ga2)};
        double e[2];
        exp_f64(x, e, c);
        return __dmul_rn(c.ghalfC, __dadd_rn(e[0], e[1]));        // ghalfC = fl(0.5*C) (exact), set by the host
    }
};

// cos_f32 of I2: Cody-Waite reduction by pi/2 in three fp32 pieces + Taylor polynomials, all explicit
// fmaf, so that the value is bit-identical to the CPU statement of the same recipe (valid |a| <= 128).
__device__ __forceinline__ float cos_f32(float a)
{
    const float qf = rintf(__fmul_rn(a, 0x1.45f306p-1f));          // rnd32(2/pi)
    float r = __fmaf_rn(qf, -0x1.921fb6p+0f, a);                    // rnd32(pi/2)
    r = __fmaf_rn(qf, 0x1.777a5cp-25f, r);                          // -rnd32(pi/2 - C1)
    r = __fmaf_rn(qf, 0x1.ee59dap-50f, r);                          // -rnd32(pi/2 - C1 - C2)
    const float z = __fmul_rn(r, r);
    float pc = -0x1.27e4fcp-22f;                                    // -1/10!
    pc = __fmaf_rn(pc, z, 0x1.a01a02p-16f);                         //  1/8!
    pc = __fmaf_rn(pc, z, -0x1.6c16c2p-10f);                        // -1/6!
    pc = __fmaf_rn(pc, z, 0x1.555556p-5f);                          //  1/4!
    pc = __fmaf_rn(pc, z, -0.5f);
    pc = __fmaf_rn(pc, z, 1.0f);
    float ps = -0x1.ae6456p-26f;                                    // -1/11!
    ps = __fmaf_rn(ps, z, 0x1.71de3ap-19f);                         //  1/9!
    ps = __fmaf_rn(ps, z, -0x1.a01a02p-13f);                        // -1/7!
    ps = __fmaf_rn(ps, z, 0x1.111112p-7f);                          //  1/5!
    ps = __fmaf_rn(ps, z, -0x1.555556p-3f);                         // -1/3!
    const float sn = __fmaf_rn(__fmul_rn(z, r), ps, r);
    const int q = static_cast<int>(qf) & 3;
    const float v = (q & 1) ? sn : pc;
    return (q == 1 || q == 2) ? -v : v;
}

struct GenzOscPeak {         // I2, BASELINE.json configs[3], fp32 per-event arithmetic
    using real = float;
    static constexpr int kId = 2;
    static constexpr bool kU32 = false;
    static constexpr bool kHasCut = false;   // true: f = 0 for events the integrand's cuts reject
    float arg, Q;
    __device__ __forceinline__ void begin(const IntegrandConsts& c) { arg = c.zphi; Q = 1.0f; }
    __device__ __forceinline__ void coord(int k, float x, const IntegrandConsts& c)
    {
        arg = __fmaf_rn(c.zc[k], x, arg);
        const float dx = __fsub_rn(x, 0.5f);
        const float pk = __fmaf_rn(dx, dx, c.zw[k]);
        Q = __fmul_rn(Q, pk);
    }
    __device__ __forceinline__ bool precheck(const IntegrandConsts&) const { return true; }
    __device__ __forceinline__ float end(const IntegrandConsts&, int) const
    {
        return __fdiv_rn(cos_f32(arg), Q);
    }
};

struct Lo2to2 {              // I3, BASELINE.json configs[4], dim = 3: (v1, v2, v3)
    using real = double;
    static constexpr int kId = 3;
    static constexpr bool kU32 = false;
    static constexpr bool kHasCut = true;   // true: f = 0 for events the integrand's cuts reject
    double v[3];
    __device__ __forceinline__ void begin(const IntegrandConsts&) {}
    __device__ __forceinline__ void coord(int k, double x, const IntegrandConsts&)
    {
        if (k == 0) v[0] = x; else if (k == 1) v[1] = x; else v[2] = x;
    }
    // the cuts, on exactly rounded quantities so that the selection is bit-reproducible (reading R15)
    __device__ __forceinline__ bool precheck(const IntegrandConsts& c) const
    {
        const double cth = __fma_rn(2.0, v[2], -1.0);
        return (__dadd_rn(v[0], v[1]) < 1.0) && (fabs(cth) < c.hcut);
    }
    // value for an event that passed precheck().  The definition (I3: g(x1) g(x2) ME flux Jac with shat = x1 x2 s)
    // is evaluated in the algebraically reduced form the reading allows ("the GPU may re-associate /
    // cancel shat"): shat cancels in ME = (shat^2 + uhat^2)/that^2 = (4 + (1+c)^2)/(1-c)^2 and in
    // flux Jac = L^2/s, and the two PDF exponentials merge: 3 exp + 1 division instead of 4 + 2.  The value differs
    // from the literal evaluation order by rounding only (a few ulp; the tests allow 2e-14).
    __device__ __forceinline__ double end(const IntegrandConsts& c, int) const
    {
        const double v1 = v[0], v2 = v[1], v3 = v[2];
        const double L = c.hL;
        const double cth = __fma_rn(2.0, v3, -1.0);
        const double ax[3] = {__dmul_rn(v1, L), __dmul_rn(v2, L), __dmul_rn(-c.ha, __dmul_rn(__dadd_rn(v1, v2), L))};
        double ex[3];
        exp_f64(ax, ex, c);
        const double x1 = ex[0], x2 = ex[1], e12 = ex[2];                                  // e12 = x1^-a x2^-a
        const double y12 = __dmul_rn(__dsub_rn(1.0, x1), __dsub_rn(1.0, x2));
        const double y2 = __dmul_rn(y12, y12);
        const double y5 = __dmul_rn(__dmul_rn(y2, y2), y12);                              // ((1-x1)(1-x2))^5
        const double opc = __dadd_rn(1.0, cth), omc = __dsub_rn(1.0, cth);
        const double ME = __ddiv_rn(__fma_rn(opc, opc, 4.0), __dmul_rn(omc, omc));
        return __dmul_rn(__dmul_rn(__dmul_rn(e12, y5), ME), c.hLLs);
    }
};

// Four-point Lagrange (cubic) interpolation of a table with knots uniform in ln x: x = tau^v, knot j at
// v_j = 1 - j/(M-1).  u = (1-v)(M-1), j = floor(u) clamped to [1, M-3], s = u - j,
//   g = ((w0 G[j-1] + w1 G[j]) + w2 G[j+1]) + w3 G[j+2],  w0 = -s(s-1)(s-2)/6, w1 = (s+1)(s-1)(s-2)/2,
//   w2 = -(s+1)s(s-2)/2, w3 = (s+1)s(s-1)/6 -- plain products and sums in this order (no contraction), so
// the value is bit-identical to the CPU statement of the same recipe.  The four loads are L1/L2-resident global
// reads (the table is a few KB): this is the PDFFlow-style gather of PAPER.md:L33, L49.
__device__ __forceinline__ double tab_interp(const double* __restrict__ G, int M, double v)
{
    const double u = __dmul_rn(__dsub_rn(1.0, v), static_cast<double>(M - 1));
    int j = static_cast<int>(floor(u));
    j = j < 1 ? 1 : (j > M - 3 ? M - 3 : j);
    const double s = __dsub_rn(u, static_cast<double>(j));
    const double sp = __dadd_rn(s, 1.0), sm1 = __dsub_rn(s, 1.0), sm2 = __dsub_rn(s, 2.0);
    const double w0 = __ddiv_rn(-__dmul_rn(__dmul_rn(s, sm1), sm2), 6.0);
    const double w1 = __ddiv_rn(__dmul_rn(__dmul_rn(sp, sm1), sm2), 2.0);
    const double w2 = __ddiv_rn(-__dmul_rn(__dmul_rn(sp, s), sm2), 2.0);
    const double w3 = __ddiv_rn(__dmul_rn(__dmul_rn(sp, s), sm1), 6.0);
    const double g0 = __ldg(G + j - 1), g1 = __ldg(G + j), g2 = __ldg(G + j + 1), g3 = __ldg(G + j + 2);
    return __dadd_rn(__dadd_rn(__dadd_rn(__dmul_rn(w0, g0), __dmul_rn(w1, g1)), __dmul_rn(w2, g2)), __dmul_rn(w3, g3));
}

struct Lo2to2Tab : Lo2to2 {  // NEXT-4: lo_2to2 with the PDF g(x) interpolated from a table (id 6)
    static constexpr int kId = 6;
    // f = g(x1) g(x2) ME flux Jac in the reduced form of Lo2to2::end (shat cancels): g1 g2 (4+(1+c)^2)/(1-c)^2 L^2/s
    __device__ __forceinline__ double end(const IntegrandConsts& c, int) const
    {
        const double cth = __fma_rn(2.0, v[2], -1.0);
        const double g1 = tab_interp(c.tab, c.ntab, v[0]);
        const double g2 = tab_interp(c.tab, c.ntab, v[1]);
        const double opc = __dadd_rn(1.0, cth), omc = __dsub_rn(1.0, cth);
        const double ME = __ddiv_rn(__fma_rn(opc, opc, 4.0), __dmul_rn(omc, omc));
        return __dmul_rn(__dmul_rn(__dmul_rn(g1, g2), ME), c.hLLs);
    }
};

template <typename Real>
struct ToySum {              // I4: tf.reduce_sum(xarr, axis=1)
    using real = Real;
    static constexpr int kId = 4;
    static constexpr bool kU32 = false;
    static constexpr bool kHasCut = false;   // true: f = 0 for events the integrand's cuts reject
    Real f;
    __device__ __forceinline__ void begin(const IntegrandConsts&) { f = Real(0); }
    __device__ __forceinline__ void coord(int, Real x, const IntegrandConsts&)
    {
        if constexpr (sizeof(Real) == 8) f = __dadd_rn(f, x); else f = __fadd_rn(f, x);
    }
    __device__ __forceinline__ bool precheck(const IntegrandConsts&) const { return true; }
    __device__ __forceinline__ Real end(const IntegrandConsts&, int) const { return f; }
};

// The same fp64 integrand driven by the 32-bit-uniform stream (VEGAS_FP64_U32).
template <class F>
struct U32 : F {
    static_assert(sizeof(typename F::real) == 8, "U32 wraps fp64 integrands");
    static constexpr bool kU32 = true;
};

// ------------------------------------------------------------------------------------------------
// One event, S1-S4.  D = compile-time dimension (0: run-time a.dim), NB = compile-time bin count (0:
// run-time a.nbins).  `tab` points to the staged table in shared memory, cell (k, i) at
// tab[(k*N + i) * TSTRIDE + toff] (TSTRIDE/toff implement lane-replicated bank-conflict-free copies).
// bins[] receives the d bin indices.  Returns wf = (double)J * (double)f.
// ------------------------------------------------------------------------------------------------
// event_front: S1 + S2 + the per-coordinate part of S3.  Leaves the integrand's accumulated state in
// `integrand` and returns J.  The table is either the staged copy in shared memory (TCELL > 0: `tab_smem` is the
// 32-bit shared address of this lane's copy of cell 0 and cells are TCELL bytes apart) or the master table in global
// memory (TCELL == 0, the parity hook).
template <class F, int D, int NB, int TCELL, class BinSink>
__device__ __forceinline__ typename F::real event_front(const IterArgs& a, uint32_t it, uint32_t e_lo, const void* tab_gmem,
                                                        uint32_t tab_smem, BinSink&& sink, F& integrand)
{
    using real = typename F::real;
    constexpr bool kF64 = (sizeof(real) == 8);
    const int d = D ? D : a.dim;
    const uint32_t N = NB ? static_cast<uint32_t>(NB) : static_cast<uint32_t>(a.nbins);
    integrand.begin(a.ic);
    real J = real(1);
    uint32_t r[4] = {0u, 0u, 0u, 0u};
    const real Nr = static_cast<real>(N);
#pragma unroll
    for (int k = 0; k < (D ? D : kMaxDim); ++k) {
        if (!D && k >= d) break;
        int i; real frac;
        if constexpr (kF64 && !F::kU32) {                // 52 bits of two words per coordinate
            if ((k & 1) == 0) philox4x32_10(e_lo, a.e_hi, it, static_cast<uint32_t>(k >> 1), a, r);
            const uint32_t w_lo = (k & 1) ? r[2] : r[0], w_hi = (k & 1) ? r[3] : r[1];
            bin_frac64(w_lo, w_hi, N, i, frac);
        } else {                                         // one 32-bit word per coordinate, four per Philox block
            if ((k & 3) == 0) philox4x32_10(e_lo, a.e_hi, it, static_cast<uint32_t>(k >> 2), a, r);
            const uint32_t w = ((k & 3) == 0) ? r[0] : ((k & 3) == 1) ? r[1] : ((k & 3) == 2) ? r[2] : r[3];
            if constexpr (kF64) bin_frac64_u32(w, N, i, frac); else bin_frac32(w, N, i, frac);
        }
        real lo, wd;
        if constexpr (TCELL > 0)                         // k*N*TCELL is an immediate when D and NB are compile-time
            lds_cell(tab_smem + static_cast<uint32_t>(k) * N * TCELL + static_cast<uint32_t>(i) * TCELL, lo, wd);
        else
            ldg_cell(tab_gmem, k * static_cast<int>(N) + i, lo, wd);
        real x, g;
        if constexpr (kF64) { x = __fma_rn(frac, wd, lo); g = __dmul_rn(Nr, wd); J = (k == 0) ? g : __dmul_rn(J, g); }
        else { x = __fmaf_rn(frac, wd, lo); g = __fmul_rn(Nr, wd); J = (k == 0) ? g : __fmul_rn(J, g); }
        sink(k, i, x);
        integrand.coord(k, x, a.ic);
    }
    return J;
}

// One whole event, S1-S4: returns wf = (double)J * (double)f.
template <class F, int D, class BinSink>
__device__ __forceinline__ double process_event(const IterArgs& a, uint32_t e_lo, const void* tab_gmem,
                                                BinSink&& sink, typename F::real& J_out,
                                                typename F::real& f_out, bool& pass)
{
    using real = typename F::real;
    F integrand;
    const real J = event_front<F, D, 0, 0>(a, a.iteration, e_lo, tab_gmem, 0u, sink, integrand);
    pass = integrand.precheck(a.ic);
    const real f = pass ? integrand.end(a.ic, D ? D : a.dim) : real(0);
    J_out = J;
    f_out = f;
    return __dmul_rn(static_cast<double>(J), static_cast<double>(f));   // S4
}

}  // namespace vegas
