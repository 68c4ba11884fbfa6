// vegas_api.cu -- C ABI of libvegas_b200.so (include/vegas_b200.h): host driver of the Vegas hot path.
//
// The host side only validates arguments, lays out the caller's device workspace, cuts an iteration
// into launches (a8, PAPER.md:L57-L65 `events_limit`) and enqueues kernels on the caller's stream.
// Every step S1-S7 runs in the kernels of vegas_kernels.cuh; there is no CPU fallback.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <type_traits>

#include <cuda_runtime.h>

#include "../../include/vegas_b200.h"
#include "vegas_kernels.cuh"
#include "vegas_rtc.h"

namespace {

using namespace vegas;

constexpr int kMaxTable = 4096;         // doubles of integrand data (tabulated PDF)
constexpr int kRing = 64;               // (I, sigma) entries logged on the device between two reads of a graph run
constexpr int kStepsPerGraph = 16;      // consecutive single-launch steps captured into one CUDA graph (vegas_run_integration)
constexpr int kEvPool = 64;             // CUDA-event pairs kept for the most recent iterations' device times
constexpr int kLanes = 128;             // internal streams the launches of one iteration are dealt to (a8): as many as the
                                        // device runs kernels concurrently
constexpr double kCtaOverheadEvents = 3.0;   // a CTA's prologue + flush + launch cost, in events per thread (measured on
                                        // configs[1]: ~6 us against 2.2 us per event and thread of a full SM)
constexpr double kOversubscribe = 1.15;  // CTAs in flight aimed at, relative to the CTA slots, when launches are tiny (plan_launches)
constexpr int kLaneSlots = 2048;        // upper bound on the iterate grid (CTAs) = slots of a lane's region
constexpr int kMaxSlots = 8 * kLaneSlots;   // lanes x (largest grid among the launches) never exceeds this
constexpr size_t kStaticSmemReserve = 1024;   // the opt-in shared-memory limit covers static + dynamic: room for the kernels' few static words
constexpr int kPartHeader = 8;          // doubles in front of H: S1.hi, S1.lo, S2.hi, S2.lo, npass, pad[3] (vegas_partials)
constexpr uint32_t kDebugChunk = 4096;  // events per pass of vegas_debug_events through the workspace's scratch region
constexpr uint64_t kMaxLaunches = uint64_t(1) << 20;   // sanity bound on the launches of one iteration
constexpr uint64_t kGraphMinLaunches = 16;   // vegas_iterate replays a captured graph from this many launches on
constexpr double kPi = 0x1.921fb54442d18p+1;   // fl64(pi)

thread_local char g_err[4096] = "";

int fail(int code, const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

#define CUDA_TRY(expr)                                                                               \
    do {                                                                                             \
        cudaError_t e_ = (expr);                                                                     \
        if (e_ != cudaSuccess)                                                                       \
            return fail(VEGAS_ECUDA, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e_), __FILE__, __LINE__); \
    } while (0)

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// ---- device workspace layout (all offsets 256-byte aligned) -------------------------------------
struct Layout {
    size_t edges, new_edges, table, zero_begin, part, hist, slots, npass, zero_end, result, flags, status, dev_iter, ring, idata,
        scratch, total;
};

Layout make_layout(int dim, int nbins)
{
    Layout L{};
    const size_t cells = static_cast<size_t>(dim) * nbins, nedges = static_cast<size_t>(dim) * (nbins + 1);
    size_t o = 0;
    L.edges = o;      o = align_up(o + nedges * 8, 256);
    L.new_edges = o;  o = align_up(o + nedges * 8, 256);
    L.table = o;      o = align_up(o + cells * 16, 256);
    L.zero_begin = o;                                   // [partials header | hist | slots | npass] is cleared by one memset
    L.part = o;                                         // the unreduced partials of one iteration, contiguous (NEXT-2):
    L.hist = o + kPartHeader * 8;                       // 8-double header, then H[dim][nbins]
    o = align_up(L.hist + cells * 8, 256);
    L.slots = o;      o = align_up(o + static_cast<size_t>(kMaxSlots) * 32, 256);
    L.npass = o;      o = align_up(o + 8, 256);
    L.zero_end = o;
    L.result = o;     o = align_up(o + 64, 256);
    L.flags = o;      o = align_up(o + kMaxDim * 4, 256);
    L.status = o;     o = align_up(o + 16, 256);                   // refine: rejected count, ticket counter, latest outcome
    L.dev_iter = o;   o = align_up(o + 4, 256);                    // iteration counter of CUDA-graph replays
    L.ring = o;       o = align_up(o + (static_cast<size_t>(kRing) * 3 + 1) * 8, 256);   // their (I, sigma, time stamp) log + start stamp
    L.idata = o;      o = align_up(o + static_cast<size_t>(kMaxTable) * 8, 256);     // integrand data (vegas_set_table)
    L.scratch = o;    o = align_up(o + static_cast<size_t>(kDebugChunk) * (static_cast<size_t>(dim) * 12 + 32), 256);   // vegas_debug_events
    L.total = o;
    return L;
}

// ---- compiled kernel instances -------------------------------------------------------------------
using LaunchFn = cudaError_t (*)(const IterArgs&, int grid, int threads, size_t smem, cudaStream_t);
using DebugFn = cudaError_t (*)(const IterArgs&, int grid, int threads, cudaStream_t, int32_t*, double*, double*,
                                double*, double*, int32_t*);
using AttrFn = cudaError_t (*)(int smem_bytes);
using OccFn = cudaError_t (*)(int* ctas, int threads, size_t smem);

struct Instance {
    int integrand_id, dim /* 0 = any */, nbins /* 0 = any */, precision;
    int rs /* log2 histogram replicas, -1 = run-time */, trep /* table replicas */, max_threads;
    int def_ctas, def_threads;       // default launch shape
    int queue_entry_bytes;           // per-entry bytes of the per-warp compaction queue (0: integrand has no cut)
    LaunchFn launch;
    DebugFn debug;
    AttrFn set_smem;
    OccFn occupancy;
    const void* rt_iterate;          // run-time compiled instance (vegas_create_custom): cudaKernel_t handles used
    const void* rt_debug;            // instead of the four function pointers above
};

// VEGAS_NO_PDL=1 in the environment switches programmatic dependent launch off (plain stream order)
const bool g_use_pdl = [] { const char* e = std::getenv("VEGAS_NO_PDL"); return !(e && e[0] == '1'); }();
// Cleared by enqueue_iteration around the launches of an iteration that is dealt to several stream lanes: there whole
// chains of dependent kernels would become resident and sit at griddepcontrol.wait holding shared memory and thread
// slots that other lanes' kernels need (measured on configs[2], 1e4 events per launch: 2.67 ms with the attribute,
// 2.62 ms without; 1e5 and up: no difference).  The attribute pays where launches follow one another on ONE stream.
thread_local bool t_pdl_this_launch = true;

// Launch configuration of every iterate_kernel launch: programmatic stream serialization allowed, i.e. the launch may
// begin (its shared-memory prologue, up to griddepcontrol.wait) while the kernel in front of it on the stream is still
// in its tail.  `attr` must outlive the returned configuration.
cudaLaunchConfig_t iterate_launch_config(int grid, int threads, size_t smem, cudaStream_t st, cudaLaunchAttribute* attr)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(static_cast<unsigned>(grid));
    cfg.blockDim = dim3(static_cast<unsigned>(threads));
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = (g_use_pdl && t_pdl_this_launch) ? 1 : 0;
    return cfg;
}

// One interface for compiled-in and run-time compiled instances.
cudaError_t inst_launch(const Instance* in, const IterArgs& a, int grid, int threads, size_t smem, cudaStream_t st)
{
    if (!in->rt_iterate) return in->launch(a, grid, threads, smem, st);
    void* args[] = {const_cast<IterArgs*>(&a)};
    cudaLaunchAttribute attr[1];
    const cudaLaunchConfig_t cfg = iterate_launch_config(grid, threads, smem, st, attr);
    return cudaLaunchKernelExC(&cfg, in->rt_iterate, args);
}
cudaError_t inst_debug(const Instance* in, const IterArgs& a, int grid, int threads, cudaStream_t st, int32_t* bins,
                       double* x, double* jac, double* f, double* wf, int32_t* pass)
{
    if (!in->rt_debug) return in->debug(a, grid, threads, st, bins, x, jac, f, wf, pass);
    void* args[] = {const_cast<IterArgs*>(&a), &bins, &x, &jac, &f, &wf, &pass};
    return cudaLaunchKernel(in->rt_debug, dim3(grid), dim3(threads), args, 0, st);
}
cudaError_t inst_set_smem(const Instance* in, int smem_bytes)
{
    if (!in->rt_iterate) return in->set_smem(smem_bytes);
    return cudaFuncSetAttribute(in->rt_iterate, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes);
}
cudaError_t inst_occupancy(const Instance* in, int* ctas, int threads, size_t smem)
{
    if (!in->rt_iterate) return in->occupancy(ctas, threads, smem);
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(ctas, in->rt_iterate, threads, smem);
}

template <class F, int D, int NB, int RS, int TREP, int HB, int MAXT, int MINB>
cudaError_t launch_iterate(const IterArgs& a, int grid, int threads, size_t smem, cudaStream_t st)
{
    cudaLaunchAttribute attr[1];
    const cudaLaunchConfig_t cfg = iterate_launch_config(grid, threads, smem, st, attr);
    return cudaLaunchKernelEx(&cfg, iterate_kernel<F, D, NB, RS, TREP, HB, MAXT, MINB>, a);
}
template <class F, int D>
cudaError_t launch_debug(const IterArgs& a, int grid, int threads, cudaStream_t st, int32_t* bins, double* x,
                         double* jac, double* f, double* wf, int32_t* pass)
{
    debug_events_kernel<F, D><<<grid, threads, 0, st>>>(a, bins, x, jac, f, wf, pass);
    return cudaGetLastError();
}
template <class F, int D, int NB, int RS, int TREP, int HB, int MAXT, int MINB>
cudaError_t set_smem_attr(int smem_bytes)
{
    return cudaFuncSetAttribute(iterate_kernel<F, D, NB, RS, TREP, HB, MAXT, MINB>,
                                cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes);
}
template <class F, int D, int NB, int RS, int TREP, int HB, int MAXT, int MINB>
cudaError_t query_occupancy(int* ctas, int threads, size_t smem)
{
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(ctas, iterate_kernel<F, D, NB, RS, TREP, HB, MAXT, MINB>,
                                                         threads, smem);
}

template <class F, int D>
constexpr int queue_entry_bytes()
{
    return F::kHasCut ? static_cast<int>(sizeof(F) + 8 + ((sizeof(BinPack<D>) / 4 + 1) / 2) * 8) : 0;
}

// TUNED: compile-time dim, bin count, replica counts (one per BASELINE.json configuration; the launch
// shape was chosen by the sweep recorded in DESIGN.md).  GENERIC: everything run-time.
#define VEGAS_TUNED(ID, F, D, NB, RS, TREP, HB, PREC, MAXT, CTAS, THREADS)                               \
    Instance { ID, D, NB, PREC, RS, TREP, MAXT, CTAS, THREADS, queue_entry_bytes<F, D>(), launch_iterate<F, D, NB, RS, TREP, HB, MAXT, 1>, \
               launch_debug<F, D>, set_smem_attr<F, D, NB, RS, TREP, HB, MAXT, 1>,                       \
               query_occupancy<F, D, NB, RS, TREP, HB, MAXT, 1>, nullptr, nullptr }
#define VEGAS_GENERIC(ID, F, D, PREC)                                                                    \
    Instance { ID, D, 0, PREC, -1, 1, 1024, 2, 512, queue_entry_bytes<F, D>(), launch_iterate<F, D, 0, -1, 1, 0, 1024, 1>,   \
               launch_debug<F, D>, set_smem_attr<F, D, 0, -1, 1, 0, 1024, 1>,                     \
               query_occupancy<F, D, 0, -1, 1, 0, 1024, 1>, nullptr, nullptr }


const Instance kInstances[] = {
    VEGAS_TUNED(VEGAS_GAUSS_SYM, GaussSym, 4, 50, 5, 8, 4, VEGAS_FP64, 1024, 1, 1024),            // configs[0]
    VEGAS_TUNED(VEGAS_GAUSS_DOUBLE, GaussDouble, 8, 50, 5, 8, 4, VEGAS_FP64, 768, 1, 768),      // configs[1], [2]
    VEGAS_TUNED(VEGAS_GENZ_OSC_PEAK, GenzOscPeak, 20, 100, 3, 4, 0, VEGAS_FP32_EVAL, 1024, 1, 1024),  // configs[3]
    VEGAS_TUNED(VEGAS_LO_2TO2, Lo2to2, 3, 50, 5, 8, 3, VEGAS_FP64, 1024, 2, 1024),                // configs[4]
    VEGAS_TUNED(VEGAS_GAUSS_DOUBLE, U32<GaussDouble>, 8, 50, 5, 8, 4, VEGAS_FP64_U32, 768, 1, 768),   // configs[1] with 32-bit uniforms
    VEGAS_TUNED(VEGAS_LO_2TO2_TAB, Lo2to2Tab, 3, 50, 5, 8, 3, VEGAS_FP64, 1024, 2, 1024),         // NEXT-4
    VEGAS_GENERIC(VEGAS_LO_2TO2_TAB, Lo2to2Tab, 3, VEGAS_FP64),
    VEGAS_GENERIC(VEGAS_GAUSS_SYM, GaussSym, 4, VEGAS_FP64),
    VEGAS_GENERIC(VEGAS_GAUSS_DOUBLE, GaussDouble, 8, VEGAS_FP64),
    VEGAS_GENERIC(VEGAS_GENZ_OSC_PEAK, GenzOscPeak, 20, VEGAS_FP32_EVAL),
    VEGAS_GENERIC(VEGAS_LO_2TO2, Lo2to2, 3, VEGAS_FP64),
    VEGAS_GENERIC(VEGAS_TOY_SUM, ToySum<double>, 10, VEGAS_FP64),
    VEGAS_GENERIC(VEGAS_GAUSS_SYM, GaussSym, 0, VEGAS_FP64),
    VEGAS_GENERIC(VEGAS_GAUSS_DOUBLE, GaussDouble, 0, VEGAS_FP64),
    VEGAS_GENERIC(VEGAS_GENZ_OSC_PEAK, GenzOscPeak, 0, VEGAS_FP32_EVAL),
    VEGAS_GENERIC(VEGAS_TOY_SUM, ToySum<double>, 0, VEGAS_FP64),
    VEGAS_GENERIC(VEGAS_TOY_SUM, ToySum<float>, 0, VEGAS_FP32_EVAL),
    VEGAS_GENERIC(VEGAS_GAUSS_SYM, U32<GaussSym>, 0, VEGAS_FP64_U32),
    VEGAS_GENERIC(VEGAS_GAUSS_DOUBLE, U32<GaussDouble>, 0, VEGAS_FP64_U32),
    VEGAS_GENERIC(VEGAS_LO_2TO2, U32<Lo2to2>, 3, VEGAS_FP64_U32),
    VEGAS_GENERIC(VEGAS_TOY_SUM, U32<ToySum<double>>, 0, VEGAS_FP64_U32),
};

// The tuned instance for exactly (id, dim, nbins, precision), or NULL.
const Instance* find_tuned(int id, int dim, int nbins, int precision)
{
    for (const Instance& in : kInstances)
        if (in.rs >= 0 && in.integrand_id == id && in.precision == precision && in.dim == dim && in.nbins == nbins) return &in;
    return nullptr;
}

// The run-time-shaped instance: exact dimension first, then any dimension.
const Instance* find_generic(int id, int dim, int precision)
{
    for (const Instance& in : kInstances)
        if (in.rs < 0 && in.integrand_id == id && in.precision == precision && in.dim == dim) return &in;
    for (const Instance& in : kInstances)
        if (in.rs < 0 && in.integrand_id == id && in.precision == precision && in.dim == 0) return &in;
    return nullptr;
}

int expected_params(int id, int dim)
{
    switch (id) {
        case VEGAS_GAUSS_SYM: return 2;
        case VEGAS_GAUSS_DOUBLE: return 3;
        case VEGAS_GENZ_OSC_PEAK: return 1 + dim;
        case VEGAS_LO_2TO2: return 5;
        case VEGAS_TOY_SUM: return 0;
        case VEGAS_LO_2TO2_TAB: return 3;
        case VEGAS_USER: return -2;          // any count up to kMaxUserParams (checked by vegas_create_custom)
        default: return -1;
    }
}

}  // namespace

// Lets the library's other translation units (vegas_static.cu) record the message vegas_last_error() returns.  Not
// exported from the shared object.
__attribute__((visibility("hidden"))) int vegas_detail_fail(int code, const char* msg) { return fail(code, "%s", msg); }

struct vegas_ctx {
    int dim, nbins, integrand_id, precision;
    const Instance* inst;            // the instance in use (tuned or generic, chosen by apply_shape)
    const Instance* tuned;           // may be NULL
    const Instance* generic;
    cudaStream_t stream;
    unsigned char* ws;
    Layout L;
    IntegrandConsts ic;
    uint32_t iteration;
    bool have_hist, have_sums;
    int sm_count, sm_clock_khz, smem_optin;
    int ctas_per_sm, threads, rshift;            // launch shape in use
    size_t smem_bytes;
    double* h_result;        // pinned: result[8] then hist[dim*nbins]
    int* h_status;           // pinned
    double* h_ring;          // pinned: kRing (I, sigma) pairs read back from graph replays
    cudaEvent_t run_ev0, run_ev1;    // bracket a whole graph-replayed run
    cudaStream_t gstream;            // internal capturable stream the graph is captured on and replayed in
                                     // (the caller's stream may be the legacy default stream, which cannot capture)
    cudaEvent_t evA[kEvPool], evB[kEvPool];   // pair (n % kEvPool) brackets the n-th enqueued iteration
    uint64_t n_enqueued;             // iterations enqueued so far
    int refine_pending;              // refinements enqueued and not yet collected
    cudaLibrary_t rt_lib;            // vegas_create_custom: the loaded cubin and its Instance (owned)
    Instance* rt_inst;
    int n_user_params;
    int use_graph;                   // vegas_run_integration replays a captured step (vegas_use_cuda_graph)
    cudaGraphExec_t gexec;           // captured {memset, launches, finalize, refine, commit} for the key below
    cudaGraphExec_t gexec_k;         // kStepsPerGraph of them in one graph (single-launch steps only)
    uint64_t g_n, g_epl, g_seed; double g_alpha; int g_threads, g_ctas, g_rshift; const Instance* g_inst;
    cudaStream_t lane[kLanes];       // non-blocking streams: small launches of one iteration overlap on the GPU
    cudaEvent_t lane_done[kLanes], fork;
    uint64_t last_n;
    int last_launches;
    bool hist_consumed;              // the latest refinement took the histogram and no iteration ran since: a rejected
                                     // refinement gives it back (grid and H unchanged, DESIGN.md section 2 S7)
    bool last_graph;                 // the latest iteration(s) ran as graph replays of whole steps: no per-iteration events
    double last_graph_ms;            // their average device time per step
    bool shard_pending;              // vegas_iterate_shard_enqueue ran and vegas_finalize_enqueue has not yet
    bool accum_clean;                // [partials | H | slots | pass counter | ticket] are all zero on the device (after create /
                                     // reset and after every fused step, whose last CTA clears them): no memset needed
    cudaGraphExec_t igexec;          // captured {memset, launches} of one many-launch iteration (vegas_iterate) for the key below
    double ig_alpha; uint64_t ig_n, ig_first, ig_count, ig_epl, ig_seed; int ig_threads, ig_ctas, ig_rshift, ig_shard, ig_launches; const Instance* ig_inst;
};

namespace {

// Integrand constants (I0-I3), one correctly rounded host operation per step (compiled with
// -ffp-contract=off): the same statement of the constants as DESIGN.md, independent of oracle/.
int setup_integrand(vegas_ctx* c, const double* p)
{
    std::memset(&c->ic, 0, sizeof(c->ic));
    fill_exp_consts(c->ic.ec);
    switch (c->integrand_id) {
        case VEGAS_GAUSS_SYM:
        case VEGAS_GAUSS_DOUBLE: {
            const double alpha = p[0];
            const double b = alpha * std::sqrt(kPi);
            double C = 1.0;
            for (int k = 0; k < c->dim; ++k) C = C / b;
            c->ic.gC = C;
            c->ic.ghalfC = 0.5 * C;
            c->ic.ga2 = 1.0 / (alpha * alpha);
            c->ic.gmu0 = p[1];
            c->ic.gmu1 = (c->integrand_id == VEGAS_GAUSS_DOUBLE) ? p[2] : 0.0;
            return VEGAS_OK;
        }
        case VEGAS_GENZ_OSC_PEAK: {
            c->ic.zphi = static_cast<float>((2.0 * kPi) * p[0]);
            for (int k = 0; k < c->dim; ++k) {
                const float ck = static_cast<float>(p[1 + k]);
                c->ic.zc[k] = ck;
                c->ic.zw[k] = 1.0f / (ck * ck);
            }
            return VEGAS_OK;
        }
        case VEGAS_LO_2TO2: {
            if (c->dim != 3) return fail(VEGAS_EINVAL, "lo_2to2 needs dim = 3");
            if (p[4] != 5.0) return fail(VEGAS_EUNSUPPORTED, "lo_2to2: pdf_b is fixed to 5");
            const double s = p[0] * p[0];
            const double smin = p[1] * p[1];
            const double tau = smin / s;
            c->ic.hs = s;
            c->ic.hL = std::log(tau);
            c->ic.hcut = p[2];
            c->ic.ha = p[3];
            c->ic.hLLs = (c->ic.hL * c->ic.hL) / s;
            return VEGAS_OK;
        }
        case VEGAS_LO_2TO2_TAB: {
            if (c->dim != 3) return fail(VEGAS_EINVAL, "lo_2to2_tab needs dim = 3");
            const double s = p[0] * p[0];
            c->ic.hs = s;
            c->ic.hL = std::log((p[1] * p[1]) / s);
            c->ic.hcut = p[2];
            c->ic.hLLs = (c->ic.hL * c->ic.hL) / s;
            c->ic.tab = nullptr;                          // vegas_set_table
            c->ic.ntab = 0;
            return VEGAS_OK;
        }
        case VEGAS_USER:
            for (int i = 0; i < c->n_user_params; ++i) c->ic.user_params[i] = p[i];
            return VEGAS_OK;
        default: return VEGAS_OK;
    }
}

size_t iterate_smem_bytes(const vegas_ctx* c, const Instance* in, int rshift, int threads)
{
    const size_t cells = static_cast<size_t>(c->dim) * c->nbins;
    const size_t cell_bytes = (c->precision == VEGAS_FP32_EVAL) ? 8 : 16;
    return align_up(cells * (size_t(1) << rshift) * 8, 16) + align_up(cells * in->trep * cell_bytes, 16) +
           static_cast<size_t>((threads + 31) / 32) * (5 * 8 + static_cast<size_t>(in->queue_entry_bytes) * kQueueCap);
}

// Choose R = 2^rshift: the largest power of two <= 32 such that `ctas` CTAs fit in the SM's shared memory.
int pick_rshift(const vegas_ctx* c, const Instance* in, int ctas, int threads)
{
    const size_t per_sm = 228u * 1024u;
    for (int rs = 5; rs >= 0; --rs) {
        const size_t need = iterate_smem_bytes(c, in, rs, threads) + 1024;   // 1 KB reserved per CTA
        if (need * ctas <= per_sm && need <= static_cast<size_t>(c->smem_optin)) return rs;
    }
    return -1;
}

// ctas/threads <= 0: the instance's default.  rshift < 0: the tuned instance's fixed R if it can be used,
// else the largest R that fits.  A shape the tuned instance cannot take (another R, more threads than it was compiled
// for) runs on the generic one.
int apply_shape(vegas_ctx* c, int ctas, int threads, int rshift)
{
    const Instance* in = (c->tuned && (rshift < 0 || rshift == c->tuned->rs) && threads <= c->tuned->max_threads)
                             ? c->tuned : c->generic;
    if (ctas <= 0) ctas = in->def_ctas;
    if (threads <= 0) threads = in->def_threads;
    if (threads < 32 || threads > in->max_threads || (threads & 31)) return fail(VEGAS_EINVAL, "threads_per_cta %d not in 32..%d (multiple of 32)", threads, in->max_threads);
    if (ctas < 1 || ctas > 16) return fail(VEGAS_EINVAL, "ctas_per_sm %d not in 1..16", ctas);
    if (in->rs >= 0) rshift = in->rs;
    else if (rshift < 0) rshift = pick_rshift(c, in, ctas, threads);
    if (rshift < 0 || rshift > 5) return fail(VEGAS_EINVAL, "histogram of %d x %d cells does not fit in shared memory with %d CTAs/SM", c->dim, c->nbins, ctas);
    const size_t smem = iterate_smem_bytes(c, in, rshift, threads);
    if (smem > static_cast<size_t>(c->smem_optin) - kStaticSmemReserve) return fail(VEGAS_EINVAL, "needs %zu bytes of shared memory per CTA, device allows %d", smem, c->smem_optin - static_cast<int>(kStaticSmemReserve));
    // cudaFuncAttributeMaxDynamicSharedMemorySize belongs to the kernel function, not to this context: contexts that
    // share a generic instance with different shapes must not lower each other's limit, so it is always the device maximum
    CUDA_TRY(inst_set_smem(in, c->smem_optin - static_cast<int>(kStaticSmemReserve)));
    int occ = 0;
    CUDA_TRY(inst_occupancy(in, &occ, threads, smem));
    if (occ < 1) return fail(VEGAS_EINVAL, "launch shape (%d threads, %zu B smem) cannot run", threads, smem);
    if (occ < ctas) ctas = occ;
    if (ctas * c->sm_count > kLaneSlots) ctas = kLaneSlots / c->sm_count;
    c->inst = in;
    c->ctas_per_sm = ctas; c->threads = threads; c->rshift = rshift; c->smem_bytes = smem;
    return VEGAS_OK;
}

void fill_args(const vegas_ctx* c, uint64_t seed, uint64_t first, uint32_t count, IterArgs& a)
{
    a.table = c->ws + c->L.table;
    a.hist = reinterpret_cast<double*>(c->ws + c->L.hist);
    a.partials = reinterpret_cast<double*>(c->ws + c->L.part);
    a.slots = reinterpret_cast<double*>(c->ws + c->L.slots);
    a.npass = reinterpret_cast<unsigned long long*>(c->ws + c->L.npass);
    a.e_lo_first = static_cast<uint32_t>(first);
    a.e_hi = static_cast<uint32_t>(first >> 32);
    a.count = count;
    a.iteration = c->iteration;
    a.iter_ptr = nullptr;
    a.ticket = nullptr; a.total_ctas = 0; a.slots0 = nullptr; a.fin_lanes = 0; a.fin_stride = 0; a.fin_used = 0;
    a.n_events = 0; a.result = nullptr; a.dev_iter = nullptr; a.ring = nullptr; a.ring_len = 0;
    const uint32_t k0 = static_cast<uint32_t>(seed), k1 = static_cast<uint32_t>(seed >> 32);
    for (int r = 0; r < 10; ++r) {
        a.rk0[r] = k0 + static_cast<uint32_t>(r) * 0x9E3779B9u;
        a.rk1[r] = k1 + static_cast<uint32_t>(r) * 0xBB67AE85u;
    }
    a.refine_alpha = -1.0;
    a.edges = reinterpret_cast<double*>(c->ws + c->L.edges);
    a.new_edges = reinterpret_cast<double*>(c->ws + c->L.new_edges);
    a.status = reinterpret_cast<int*>(c->ws + c->L.status);
    a.precision = c->precision == VEGAS_FP32_EVAL ? 1 : 0;
    a.smem_bytes = static_cast<int>(c->smem_bytes);
    a.dim = c->dim;
    a.nbins = c->nbins;
    a.rshift = c->rshift;
    a.ic = c->ic;
}

bool create_event_pool(vegas_ctx* c)
{
    for (int i = 0; i < kEvPool; ++i)
        if (cudaEventCreate(&c->evA[i]) != cudaSuccess || cudaEventCreate(&c->evB[i]) != cudaSuccess) return false;
    return true;
}

bool create_lanes(vegas_ctx* c)
{
    for (int i = 0; i < kLanes; ++i)
        if (cudaStreamCreateWithFlags(&c->lane[i], cudaStreamNonBlocking) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->lane_done[i], cudaEventDisableTiming) != cudaSuccess)
            return false;
    return true;
}

int build_table(vegas_ctx* c, int uniform)
{
    build_table_kernel<<<c->dim, 128, 0, c->stream>>>(reinterpret_cast<double*>(c->ws + c->L.edges),
                                                      c->ws + c->L.table, c->nbins, c->precision == VEGAS_FP32_EVAL ? 1 : 0, uniform);
    CUDA_TRY(cudaGetLastError());
    return VEGAS_OK;
}

}  // namespace

// =================================================================================================
// extern "C" entry points (documented in include/vegas_b200.h)
// =================================================================================================
extern "C" {

const char* vegas_last_error(void) { return g_err; }

size_t vegas_workspace_bytes(int dim, int nbins)
{
    if (dim < 1 || dim > kMaxDim || nbins < 2 || nbins > 4095) return 0;
    return make_layout(dim, nbins).total;
}

static int create_common(vegas_ctx** out, int dim, int nbins, int integrand_id, const double* params, int n_params,
                         int precision, void* dev_workspace, size_t workspace_bytes, void* cuda_stream,
                         const Instance* rt_inst);

int vegas_create(vegas_ctx** out, int dim, int nbins, int integrand_id, const double* params, int n_params,
                 int precision, void* dev_workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (integrand_id == VEGAS_USER) return fail(VEGAS_EINVAL, "user integrands are created with vegas_create_custom");
    return create_common(out, dim, nbins, integrand_id, params, n_params, precision, dev_workspace, workspace_bytes,
                         cuda_stream, nullptr);
}

// rt_inst != NULL: a run-time compiled instance (vegas_create_custom) replaces the table lookup.
static int create_common(vegas_ctx** out, int dim, int nbins, int integrand_id, const double* params, int n_params,
                         int precision, void* dev_workspace, size_t workspace_bytes, void* cuda_stream,
                         const Instance* rt_inst)
{
    if (!out) return fail(VEGAS_EINVAL, "out is NULL");
    *out = nullptr;
    if (dim < 1 || dim > kMaxDim) return fail(VEGAS_EINVAL, "dim %d not in 1..%d", dim, kMaxDim);
    if (precision != VEGAS_FP64 && precision != VEGAS_FP32_EVAL && precision != VEGAS_FP64_U32) return fail(VEGAS_EINVAL, "precision %d unknown", precision);
    const int max_bins = (precision == VEGAS_FP32_EVAL) ? 511 : 4095;     // m*N must be exact (S2)
    if (nbins < 2 || nbins > max_bins) return fail(VEGAS_EINVAL, "nbins %d not in 2..%d", nbins, max_bins);
    const int need = expected_params(integrand_id, dim);
    if (need == -1) return fail(VEGAS_EUNSUPPORTED, "integrand_id %d unknown", integrand_id);
    if (need == -2) { if (n_params < 0 || n_params > kMaxUserParams || (n_params > 0 && !params)) return fail(VEGAS_EINVAL, "a user integrand takes 0..%d params", kMaxUserParams); }
    else if (n_params != need || (need > 0 && !params)) return fail(VEGAS_EINVAL, "integrand %d with dim %d takes %d params, got %d", integrand_id, dim, need, n_params);
    const Instance* tuned = rt_inst ? nullptr : find_tuned(integrand_id, dim, nbins, precision);
    const Instance* inst = rt_inst ? rt_inst : find_generic(integrand_id, dim, precision);
    if (!inst) return fail(VEGAS_EUNSUPPORTED, "no compiled kernel for integrand %d, dim %d, precision %d", integrand_id, dim, precision);
    if (!dev_workspace) return fail(VEGAS_EINVAL, "dev_workspace is NULL");
    if (reinterpret_cast<uintptr_t>(dev_workspace) & 255u) return fail(VEGAS_EINVAL, "dev_workspace must be 256-byte aligned");
    const Layout L = make_layout(dim, nbins);
    if (workspace_bytes < L.total) return fail(VEGAS_ENOMEM, "workspace of %zu bytes, need %zu", workspace_bytes, L.total);

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        (void)cudaGetLastError();
        return fail(VEGAS_ECUDA, "no CUDA device (there is no CPU fallback)");
    }
    vegas_ctx* c = new (std::nothrow) vegas_ctx();
    if (!c) return fail(VEGAS_ENOMEM, "host allocation failed");
    c->dim = dim; c->nbins = nbins; c->integrand_id = integrand_id; c->precision = precision;
    c->inst = inst; c->tuned = tuned; c->generic = inst;
    c->stream = static_cast<cudaStream_t>(cuda_stream);
    c->ws = static_cast<unsigned char*>(dev_workspace);
    c->L = L;
    c->iteration = 0; c->have_hist = false; c->have_sums = false;
    c->h_result = nullptr; c->h_status = nullptr; c->h_ring = nullptr; c->run_ev0 = nullptr; c->run_ev1 = nullptr; c->gstream = nullptr; c->fork = nullptr; c->n_enqueued = 0; c->refine_pending = 0; c->use_graph = 1; c->gexec = nullptr; c->gexec_k = nullptr;
    for (int i = 0; i < kEvPool; ++i) { c->evA[i] = nullptr; c->evB[i] = nullptr; }
    for (int i = 0; i < kLanes; ++i) { c->lane[i] = nullptr; c->lane_done[i] = nullptr; }
    c->last_n = 0; c->last_launches = 0; c->rt_lib = nullptr; c->rt_inst = nullptr;
    c->hist_consumed = false; c->last_graph = false; c->last_graph_ms = 0.0; c->shard_pending = false; c->igexec = nullptr;
    c->accum_clean = false;
    c->n_user_params = n_params;
    int rc = setup_integrand(c, params);
    if (rc != VEGAS_OK) { delete c; return rc; }

    auto cleanup = [&](int code) { vegas_destroy(c); return code; };
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess)
        return cleanup(fail(VEGAS_ECUDA, "cudaGetDeviceProperties failed"));
    if (prop.major != 10 || prop.minor != 0)             // the library carries sm_100a SASS only (no PTX)
        return cleanup(fail(VEGAS_EUNSUPPORTED, "device sm_%d%d: this library is built for sm_100a (B200) only", prop.major, prop.minor));
    c->sm_count = prop.multiProcessorCount;
    c->smem_optin = static_cast<int>(prop.sharedMemPerBlockOptin);
    int khz = 0;
    cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev);
    c->sm_clock_khz = khz;
    if (cudaHostAlloc(reinterpret_cast<void**>(&c->h_result), (8 + static_cast<size_t>(dim) * nbins) * sizeof(double), cudaHostAllocDefault) != cudaSuccess ||
        cudaHostAlloc(reinterpret_cast<void**>(&c->h_status), 64, cudaHostAllocDefault) != cudaSuccess ||
        cudaHostAlloc(reinterpret_cast<void**>(&c->h_ring), (kRing * 3 + 1) * 8, cudaHostAllocDefault) != cudaSuccess ||
        cudaEventCreate(&c->run_ev0) != cudaSuccess || cudaEventCreate(&c->run_ev1) != cudaSuccess ||
        cudaStreamCreateWithFlags(&c->gstream, cudaStreamNonBlocking) != cudaSuccess ||
        !create_event_pool(c) ||
        cudaEventCreateWithFlags(&c->fork, cudaEventDisableTiming) != cudaSuccess || !create_lanes(c))
        return cleanup(fail(VEGAS_ECUDA, "pinned host buffer / event creation failed: %s", cudaGetErrorString(cudaGetLastError())));
    rc = apply_shape(c, 0, 0, -1);
    if (rc != VEGAS_OK && c->tuned) { c->tuned = nullptr; rc = apply_shape(c, 0, 0, -1); }
    if (rc != VEGAS_OK) rc = apply_shape(c, 1, 512, -1);
    if (rc != VEGAS_OK) return cleanup(rc);
    if (cudaMemsetAsync(c->ws, 0, L.total, c->stream) != cudaSuccess) return cleanup(fail(VEGAS_ECUDA, "workspace memset failed"));
    rc = build_table(c, 1);
    if (rc != VEGAS_OK) return cleanup(rc);
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return cleanup(fail(VEGAS_ECUDA, "create: %s", cudaGetErrorString(cudaGetLastError())));
    c->accum_clean = true;                               // the whole workspace was just zeroed
    *out = c;
    return VEGAS_OK;
}

int vegas_create_custom(vegas_ctx** out, int dim, int nbins, const char* source, const double* params, int n_params,
                        int precision, void* dev_workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (!out) return fail(VEGAS_EINVAL, "out is NULL");
    *out = nullptr;
    if (!source) return fail(VEGAS_EINVAL, "source is NULL");
    if (dim < 1 || dim > kMaxDim) return fail(VEGAS_EINVAL, "dim %d not in 1..%d", dim, kMaxDim);
    if (precision != VEGAS_FP64 && precision != VEGAS_FP64_U32) return fail(VEGAS_EINVAL, "user integrands are fp64: precision VEGAS_FP64 or VEGAS_FP64_U32");
    if (n_params < 0 || n_params > kMaxUserParams || (n_params > 0 && !params)) return fail(VEGAS_EINVAL, "a user integrand takes 0..%d params", kMaxUserParams);
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        (void)cudaGetLastError();
        return fail(VEGAS_ECUDA, "no CUDA device (there is no CPU fallback)");
    }
    vegas_rtc_result r;
    std::string log;
    int rc = vegas_rtc_compile(dim, precision, source, &r, &log);
    if (rc != VEGAS_OK) return fail(rc, "run-time compilation of the user integrand failed:\n%s", log.c_str());
    Instance* in = new (std::nothrow) Instance{VEGAS_USER, dim, 0, precision, -1, 1, 1024, 2, 512, 0, nullptr, nullptr,
                                               nullptr, nullptr, reinterpret_cast<const void*>(r.iterate),
                                               reinterpret_cast<const void*>(r.debug)};
    if (!in) { cudaLibraryUnload(r.library); return fail(VEGAS_ENOMEM, "host allocation failed"); }
    rc = create_common(out, dim, nbins, VEGAS_USER, params, n_params, precision, dev_workspace, workspace_bytes,
                       cuda_stream, in);
    if (rc != VEGAS_OK) { delete in; cudaLibraryUnload(r.library); return rc; }
    (*out)->rt_lib = r.library;
    (*out)->rt_inst = in;
    return VEGAS_OK;
}

void vegas_destroy(vegas_ctx* c)
{
    if (!c) return;
    // asynchronous work (enqueued iterations / refinements, graph replays) may still use the pinned buffers
    if (c->gstream) cudaStreamSynchronize(c->gstream);
    for (int i = 0; i < kLanes; ++i) if (c->lane[i]) cudaStreamSynchronize(c->lane[i]);
    if (c->h_result) cudaStreamSynchronize(c->stream);
    (void)cudaGetLastError();
    if (c->h_result) cudaFreeHost(c->h_result);
    if (c->h_status) cudaFreeHost(c->h_status);
    if (c->h_ring) cudaFreeHost(c->h_ring);
    if (c->run_ev0) cudaEventDestroy(c->run_ev0);
    if (c->run_ev1) cudaEventDestroy(c->run_ev1);
    if (c->gstream) cudaStreamDestroy(c->gstream);
    for (int i = 0; i < kEvPool; ++i) {
        if (c->evA[i]) cudaEventDestroy(c->evA[i]);
        if (c->evB[i]) cudaEventDestroy(c->evB[i]);
    }
    if (c->gexec) cudaGraphExecDestroy(c->gexec);
    if (c->gexec_k) cudaGraphExecDestroy(c->gexec_k);
    if (c->igexec) cudaGraphExecDestroy(c->igexec);
    if (c->rt_lib) cudaLibraryUnload(c->rt_lib);
    delete c->rt_inst;
    if (c->fork) cudaEventDestroy(c->fork);
    for (int i = 0; i < kLanes; ++i) {
        if (c->lane[i]) cudaStreamDestroy(c->lane[i]);
        if (c->lane_done[i]) cudaEventDestroy(c->lane_done[i]);
    }
    delete c;
}

int vegas_set_launch_shape(vegas_ctx* c, int ctas_per_sm, int threads_per_cta)
{
    if (!c) return fail(VEGAS_EINVAL, "ctx is NULL");
    return apply_shape(c, ctas_per_sm, threads_per_cta, -1);
}

int vegas_set_hist_replicas(vegas_ctx* c, int replicas)
{
    if (!c) return fail(VEGAS_EINVAL, "ctx is NULL");
    int rs = -1;
    if (replicas > 0) {
        for (rs = 0; rs <= 5 && (1 << rs) != replicas; ++rs) {}
        if (rs > 5) return fail(VEGAS_EINVAL, "replicas must be a power of two in 1..32");
    }
    return apply_shape(c, c->ctas_per_sm, c->threads, rs);
}

int vegas_get_launch_shape(const vegas_ctx* c, int* ctas_per_sm, int* threads_per_cta, int* hist_replicas,
                           size_t* smem_bytes)
{
    if (!c) return fail(VEGAS_EINVAL, "ctx is NULL");
    if (ctas_per_sm) *ctas_per_sm = c->ctas_per_sm;
    if (threads_per_cta) *threads_per_cta = c->threads;
    if (hist_replicas) *hist_replicas = 1 << c->rshift;
    if (smem_bytes) *smem_bytes = c->smem_bytes;
    return VEGAS_OK;
}

int vegas_device_info(const vegas_ctx* c, int* sm_count, int* sm_clock_khz)
{
    if (!c) return fail(VEGAS_EINVAL, "ctx is NULL");
    if (sm_count) *sm_count = c->sm_count;
    if (sm_clock_khz) *sm_clock_khz = c->sm_clock_khz;
    return VEGAS_OK;
}

// How the kernels of one iteration get their Philox iteration word and what the last CTA does with the sums.
enum IterMode {
    kPlain = 0,        // counter word in the kernel arguments; S6 in the last CTA
    kGraphStep = 1,    // captured whole step (vegas_run_integration): counter in device memory, S6 logs (I, sigma) to the
                       // ring and advances the counter
    kGraphIter = 2     // captured iteration (vegas_iterate with many launches): counter in device memory, written by the
                       // host before every replay
};

// The wave model behind the launch geometry (see enqueue_iteration): stream lanes and CTAs per launch for `count`
// events cut into launches of `epl`, with `threads` per CTA and `cta_slots` CTAs resident on the device.  Pure host
// arithmetic (exported as vegas_plan_launches for the tests and the report).
static void plan_launches(uint64_t count, uint64_t epl, int threads, int cta_slots, int* lanes_out, int* grid_out, int* extra_every_out)
{
    int lanes = 1, grid = cta_slots, extra_every = 0;
    const uint64_t n_launches = (count + epl - 1) / epl;
    if (n_launches > 1) {
        const double L = static_cast<double>(n_launches);
        const int lanes_max = n_launches < static_cast<uint64_t>(kLanes) ? static_cast<int>(n_launches) : kLanes;
        const double per_thread = static_cast<double>(epl < count ? epl : count) / static_cast<double>(threads);
        double best = 0.0;
        for (int g = 1; g <= cta_slots; ++g) {
            const double conc = std::fmin(static_cast<double>(cta_slots), static_cast<double>(lanes_max) * g);
            const double waves = std::ceil(L * g / conc);
            const double cost = waves * (kCtaOverheadEvents + per_thread / g);
            if (g == 1 || cost < best * (1.0 - 1e-9)) { best = cost; grid = g; }
        }
        lanes = lanes_max;
        while (lanes > 1 && static_cast<size_t>(lanes) * grid > static_cast<size_t>(kMaxSlots)) --lanes;
        // The device runs at most kLanes kernels at a time: when lanes x grid CTAs do not cover its CTA slots (tiny
        // launches: 128 one-CTA kernels on 148 SMs) every `extra_every`-th launch gets one CTA more, aiming at 1.15 x the
        // slots in flight (measured on configs[2] at 1e4 events per launch: 2.90 ms per 1e8 events with none, 2.77 with
        // every 6th -- exactly the slots --, 2.67 with every 3rd, 2.77 / 2.81 with every 2nd / every one).
        if (lanes * grid < cta_slots) {
            const double f = kOversubscribe * static_cast<double>(cta_slots) / (static_cast<double>(lanes) * grid) - 1.0;
            if (f > 0.02) extra_every = f >= 1.0 ? 1 : static_cast<int>(1.0 / f + 0.5);
        }
    }
    *lanes_out = lanes;
    *grid_out = grid;
    *extra_every_out = extra_every;
}

static int enqueue_iteration(vegas_ctx* c, uint64_t n_total, uint64_t first, uint64_t count, uint64_t events_per_launch,
                             uint64_t seed, int* n_kernel_launches, IterMode mode, bool shard, double fuse_alpha = -1.0);
static int iterate_common(vegas_ctx* c, uint64_t n_total, uint64_t first, uint64_t count, uint64_t events_per_launch,
                          uint64_t seed, int* n_kernel_launches, bool shard, double fuse_alpha = -1.0);

int vegas_iterate_enqueue(vegas_ctx* c, uint64_t n_events, uint64_t events_per_launch, uint64_t seed,
                          int* n_kernel_launches)
{
    return iterate_common(c, n_events, 0, n_events, events_per_launch, seed, n_kernel_launches, false);
}

// true if the refinement of this context's grid fits in the dynamic shared memory of its iterate launches
static bool can_fuse_refine(const vegas_ctx* c)
{
    return c->smem_bytes >= 4 * (static_cast<size_t>(c->nbins) + 1) * sizeof(double);
}

int vegas_step_enqueue(vegas_ctx* c, uint64_t n_events, uint64_t events_per_launch, uint64_t seed, double alpha,
                       int* n_kernel_launches)
{
    if (!c) return fail(VEGAS_EINVAL, "ctx is NULL");
    if (!(alpha >= 0.0)) return fail(VEGAS_EINVAL, "alpha must be >= 0");
    if (can_fuse_refine(c)) return iterate_common(c, n_events, 0, n_events, events_per_launch, seed, n_kernel_launches, false, alpha);
    // (a launch shape with less shared memory than one dimension's refinement needs: two kernels)
    int rc = iterate_common(c, n_events, 0, n_events, events_per_launch, seed, n_kernel_launches, false);
    if (rc == VEGAS_OK) rc = vegas_refine_enqueue(c, alpha);
    if (rc == VEGAS_OK && n_kernel_launches) *n_kernel_launches += 1;
    return rc;
}

int vegas_iterate_shard_enqueue(vegas_ctx* c, uint64_t n_total, uint64_t first, uint64_t count,
                                uint64_t events_per_launch, uint64_t seed, int* n_kernel_launches)
{
    return iterate_common(c, n_total, first, count, events_per_launch, seed, n_kernel_launches, true);
}

static int check_iteration_args(const vegas_ctx* c, uint64_t n_total, uint64_t first, uint64_t count, uint64_t epl,
                                uint64_t* n_launches)
{
    if (!c) return fail(VEGAS_EINVAL, "ctx is NULL");
    if (n_total < 2) return fail(VEGAS_EINVAL, "n_events must be >= 2");
    if (c->integrand_id == VEGAS_LO_2TO2_TAB && !c->ic.tab) return fail(VEGAS_ESTATE, "lo_2to2_tab needs vegas_set_table first");
    if (epl == 0) return fail(VEGAS_EINVAL, "events_per_launch must be > 0");
    if (n_total > (uint64_t(1) << 53)) return fail(VEGAS_EINVAL, "n_events must be <= 2^53");
    if (first > n_total || count > n_total - first) return fail(VEGAS_EINVAL, "shard [first, first + count) must lie inside [0, n_total)");
    const uint64_t e = epl < (uint64_t(1) << 31) ? epl : (uint64_t(1) << 31);
    // launches: ceil(count / epl) plus at most one more per multiple of 2^32 inside the range (a launch never straddles one)
    const uint64_t bound = (count + e - 1) / e + (count >> 32) + 2;
    if (bound > kMaxLaunches)
        return fail(VEGAS_EINVAL, "%llu events in launches of %llu: more than %llu launches for one iteration (raise events_per_launch)",
                    static_cast<unsigned long long>(count), static_cast<unsigned long long>(e), static_cast<unsigned long long>(kMaxLaunches));
    if (n_launches) *n_launches = bound;
    return VEGAS_OK;
}

__global__ void set_u32_kernel(uint32_t* p, uint32_t v) { *p = v; }

// Capture {memset, all launches} of one iteration with this geometry into a CUDA graph (kept until the key changes).
static int ensure_iter_graph(vegas_ctx* c, uint64_t n_total, uint64_t first, uint64_t count, uint64_t epl, uint64_t seed,
                             bool shard, double fuse_alpha, int* launches)
{
    if (c->igexec && c->ig_n == n_total && c->ig_first == first && c->ig_count == count && c->ig_epl == epl &&
        c->ig_seed == seed && c->ig_alpha == fuse_alpha && c->ig_shard == (shard ? 1 : 0) && c->ig_threads == c->threads && c->ig_ctas == c->ctas_per_sm &&
        c->ig_rshift == c->rshift && c->ig_inst == c->inst) {
        if (launches) *launches = c->ig_launches;
        return VEGAS_OK;
    }
    if (c->igexec) { cudaGraphExecDestroy(c->igexec); c->igexec = nullptr; }
    cudaStream_t user = c->stream;
    c->stream = c->gstream;                              // the caller's stream may be the legacy default stream (no capture)
    cudaError_t e = cudaStreamBeginCapture(c->gstream, cudaStreamCaptureModeRelaxed);
    if (e != cudaSuccess) { c->stream = user; return fail(VEGAS_ECUDA, "cudaStreamBeginCapture failed: %s", cudaGetErrorString(e)); }
    int nl = 0;
    const int rc = enqueue_iteration(c, n_total, first, count, epl, seed, &nl, kGraphIter, shard, fuse_alpha);
    cudaGraph_t graph = nullptr;
    e = cudaStreamEndCapture(c->gstream, &graph);       // always leave capture mode
    c->stream = user;
    if (rc != VEGAS_OK) { if (graph) cudaGraphDestroy(graph); return rc; }
    if (e != cudaSuccess) return fail(VEGAS_ECUDA, "cudaStreamEndCapture failed: %s", cudaGetErrorString(e));
    const cudaError_t e2 = cudaGraphInstantiate(&c->igexec, graph, 0);
    cudaGraphDestroy(graph);
    if (e2 != cudaSuccess) { c->igexec = nullptr; return fail(VEGAS_ECUDA, "cudaGraphInstantiate failed: %s", cudaGetErrorString(e2)); }
    c->ig_n = n_total; c->ig_first = first; c->ig_count = count; c->ig_epl = epl; c->ig_seed = seed; c->ig_shard = shard ? 1 : 0;
    c->ig_alpha = fuse_alpha;
    c->ig_threads = c->threads; c->ig_ctas = c->ctas_per_sm; c->ig_rshift = c->rshift; c->ig_inst = c->inst;
    c->ig_launches = nl;
    if (launches) *launches = nl;
    return VEGAS_OK;
}

// One iteration (or one shard of it) on the context's stream, bracketed by the event pair of the pool, with the
// host-side bookkeeping.  Iterations cut into many launches replay a captured graph (vegas_use_cuda_graph): the
// host's launch rate (2-2.5 us per cudaLaunchKernel) is otherwise the floor of small batches.
static int iterate_common(vegas_ctx* c, uint64_t n_total, uint64_t first, uint64_t count, uint64_t events_per_launch,
                          uint64_t seed, int* n_kernel_launches, bool shard, double fuse_alpha)
{
    uint64_t bound = 0;
    int rc = check_iteration_args(c, n_total, first, count, events_per_launch, &bound);
    if (rc != VEGAS_OK) return rc;
    const int evi = static_cast<int>(c->n_enqueued % kEvPool);
    int launches = 0;
    const uint64_t epl = events_per_launch < (uint64_t(1) << 31) ? events_per_launch : (uint64_t(1) << 31);
    if (c->use_graph && (count + epl - 1) / epl >= kGraphMinLaunches) {
        rc = ensure_iter_graph(c, n_total, first, count, events_per_launch, seed, shard, fuse_alpha, &launches);
        if (rc != VEGAS_OK) return rc;
        CUDA_TRY(cudaEventRecord(c->evA[evi], c->stream));
        c->accum_clean = false;                          // dirty from here on; clean again only if a whole fused step got out
        set_u32_kernel<<<1, 1, 0, c->stream>>>(reinterpret_cast<uint32_t*>(c->ws + c->L.dev_iter), c->iteration);
        CUDA_TRY(cudaGraphLaunch(c->igexec, c->stream));
    } else {
        CUDA_TRY(cudaEventRecord(c->evA[evi], c->stream));
        rc = enqueue_iteration(c, n_total, first, count, events_per_launch, seed, &launches, kPlain, shard, fuse_alpha);
        if (rc != VEGAS_OK) return rc;
    }
    CUDA_TRY(cudaEventRecord(c->evB[evi], c->stream));
    const bool fused = fuse_alpha >= 0.0;
    c->n_enqueued += 1;
    c->iteration += 1;
    c->have_hist = !shard && !fused;                     // a shard's H is partial until the all-reduce + vegas_finalize_enqueue;
    c->have_sums = !shard;                               // a fused step's H was consumed (and cleared) by its refinement
    c->shard_pending = shard;
    c->hist_consumed = false;
    c->accum_clean = fused;
    if (fused) c->refine_pending += 1;
    c->last_graph = false;
    c->last_n = n_total;
    c->last_launches = launches;
    if (n_kernel_launches) *n_kernel_launches = launches;
    return VEGAS_OK;
}

// Enqueue {memset, launches} of the events [first, first + count) of an iteration of n_total events.  Pure enqueue: no
// timing events, no bookkeeping (iterate_common / the graph captures do that).
static int enqueue_iteration(vegas_ctx* c, uint64_t n_total, uint64_t first, uint64_t count, uint64_t events_per_launch,
                             uint64_t seed, int* n_kernel_launches, IterMode mode, bool shard, double fuse_alpha)
{
    uint64_t bound = 0;
    const int rc0 = check_iteration_args(c, n_total, first, count, events_per_launch, &bound);
    if (rc0 != VEGAS_OK) return rc0;
    const uint64_t epl = events_per_launch < (uint64_t(1) << 31) ? events_per_launch : (uint64_t(1) << 31);
    // the accumulators are cleared by one memset -- unless the previous step was a fused one, whose last CTA left them clean
    // (a captured graph always carries the memset unless it is a fused step's: those are only replayed on clean accumulators)
    const bool fused = fuse_alpha >= 0.0;
    if (!(fused && (mode == kGraphStep || (mode == kPlain && c->accum_clean))))
        CUDA_TRY(cudaMemsetAsync(c->ws + c->L.zero_begin, 0, c->L.zero_end - c->L.zero_begin, c->stream));
    // From the first launch on the accumulators (slots, H, pass counter, ticket) are dirty, and they stay so if a launch
    // below fails: the last CTA of such a step never runs, so nothing clears them.  iterate_common sets the flag again
    // once every launch of a fused step was enqueued.  (Captures enqueue nothing: the flag describes the device.)
    if (mode == kPlain) c->accum_clean = false;
    if (n_kernel_launches) *n_kernel_launches = 0;
    if (count == 0) return VEGAS_OK;                     // an empty shard contributes zeros
    IterArgs a;
    fill_args(c, seed, 0, 0, a);
    if (mode != kPlain) a.iter_ptr = reinterpret_cast<const uint32_t*>(c->ws + c->L.dev_iter);
    const int max_grid = c->ctas_per_sm * c->sm_count;
    // Launches of one iteration are independent (global event index; the histogram and the pass counter are
    // accumulated with global reductions; each lane has its own slot region), so when an iteration is cut into
    // several launches they are dealt round-robin to kLanes internal streams forked from the caller's stream:
    // launches that do not fill the GPU overlap, and every launch's prologue/flush overlaps its neighbours'.
    const uint64_t n_launches = (count + epl - 1) / epl;
    // Launch geometry of a many-launch iteration (configs[2]): every launch gets the same grid g, chosen by a wave model.
    // With L launches of cnt events each, up to min(L, kLanes) of them in flight and S CTA slots on the device,
    // the CTAs run in ceil(L g / min(S, lanes g)) waves, each as long as one CTA: its fixed cost (zeroing and flushing
    // the shared histogram, staging the table, the launch itself: kCtaOverheadEvents events per thread) plus
    // cnt / (g threads) events per thread.  Small g amortises the fixed cost, large g evens out the last wave; the model
    // reproduces the measured times of the batch-size sweep to a few percent.
    int lanes = 1, cap_grid = max_grid, extra_every = 0;
    plan_launches(count, epl, c->threads, max_grid, &lanes, &cap_grid, &extra_every);
    if (lanes > 1) {
        CUDA_TRY(cudaEventRecord(c->fork, c->stream));
        for (int i = 0; i < lanes; ++i) CUDA_TRY(cudaStreamWaitEvent(c->lane[i], c->fork, 0));
    }
    double* slots0 = reinterpret_cast<double*>(c->ws + c->L.slots);
    // launch geometry of the whole iteration first: the sums are folded in the CTA that finishes last, so every launch
    // must know how many CTAs there are in total and how many slots each stream-lane region uses
    const uint64_t last = first + count;
    auto launch_count = [&](uint64_t at) {
        uint64_t cnt = last - at;
        if (cnt > epl) cnt = epl;
        const uint64_t to_wrap = (uint64_t(1) << 32) - (at & 0xFFFFFFFFull);    // never straddle 2^32 (e_hi uniform)
        return cnt > to_wrap ? to_wrap : cnt;
    };
    auto launch_grid = [&](uint64_t cnt, int index) {
        // one launch: spread even few events over all SMs (the CTAs' fixed costs run side by side; at least a warp of
        // events each); several launches share the GPU: never more threads than events
        const uint64_t per_cta = (n_launches == 1) ? 32u : static_cast<uint64_t>(c->threads);
        uint64_t want = (cnt + per_cta - 1) / per_cta;
        if (want < 1) want = 1;
        const int cap = cap_grid + ((extra_every > 0 && index % extra_every == 0) ? 1 : 0);
        return want < static_cast<uint64_t>(cap) ? static_cast<int>(want) : cap;
    };
    uint64_t total_ctas = 0;
    int used_grid = 0;
    {
        int index = 0;
        for (uint64_t at = first; at < last; ++index) {
            const uint64_t cnt = launch_count(at);
            const int grid = launch_grid(cnt, index);
            total_ctas += static_cast<uint64_t>(grid);
            if (grid > used_grid) used_grid = grid;
            at += cnt;
        }
    }
    if (total_ctas > 0xFFFFFFFFull) return fail(VEGAS_EINVAL, "too many launches for one iteration (raise events_per_launch)");
    a.ticket = reinterpret_cast<unsigned int*>(c->ws + c->L.npass) + 4;   // inside the region cleared by the memset
    a.total_ctas = static_cast<unsigned int>(total_ctas);
    a.slots0 = slots0;
    // slot regions: one per stream lane, used_grid slots each (lanes x used_grid <= kMaxSlots: the lane count was
    // reduced above if the wave model picked a grid too large for that)
    if (static_cast<size_t>(lanes) * used_grid > static_cast<size_t>(kMaxSlots)) return fail(VEGAS_EINVAL, "launch geometry needs more slot regions than the workspace holds");
    a.fin_lanes = lanes; a.fin_stride = used_grid; a.fin_used = used_grid;
    a.n_events = shard ? 0ull : n_total;
    a.result = reinterpret_cast<double*>(c->ws + c->L.result);
    a.dev_iter = (mode == kGraphStep) ? reinterpret_cast<uint32_t*>(c->ws + c->L.dev_iter) : nullptr;
    a.ring = (mode == kGraphStep) ? reinterpret_cast<double*>(c->ws + c->L.ring) : nullptr;
    a.ring_len = kRing;
    a.refine_alpha = fused ? fuse_alpha : -1.0;
    int launches = 0;
    struct PdlScope {                                    // programmatic dependent launch only on the single-stream path
        explicit PdlScope(bool on) { t_pdl_this_launch = on; }
        ~PdlScope() { t_pdl_this_launch = true; }
    } pdl_scope(lanes == 1);
    for (uint64_t at = first; at < last;) {
        const uint64_t cnt = launch_count(at);
        a.e_lo_first = static_cast<uint32_t>(at);
        a.e_hi = static_cast<uint32_t>(at >> 32);
        a.count = static_cast<uint32_t>(cnt);
        const int grid = launch_grid(cnt, launches);
        const int ln = launches % lanes;
        a.slots = slots0 + static_cast<size_t>(ln) * used_grid * 4;
        CUDA_TRY(inst_launch(c->inst, a, grid, c->threads, c->smem_bytes, lanes > 1 ? c->lane[ln] : c->stream));
        at += cnt;
        ++launches;
    }
    if (lanes > 1) {
        for (int i = 0; i < lanes; ++i) {
            CUDA_TRY(cudaEventRecord(c->lane_done[i], c->lane[i]));
            CUDA_TRY(cudaStreamWaitEvent(c->stream, c->lane_done[i], 0));
        }
    }
    CUDA_TRY(cudaGetLastError());
    if (n_kernel_launches) *n_kernel_launches = launches;
    return VEGAS_OK;
}

int vegas_plan_launches(uint64_t n_events, uint64_t events_per_launch, int threads_per_cta, int cta_slots, int* n_launches,
                        int* stream_lanes, int* ctas_per_launch, int* extra_cta_every)
{
    if (n_events < 1 || events_per_launch < 1 || threads_per_cta < 32 || threads_per_cta > 1024 || cta_slots < 1 || cta_slots > kLaneSlots)
        return fail(VEGAS_EINVAL, "vegas_plan_launches: n_events, events_per_launch >= 1, 32 <= threads_per_cta <= 1024, 1 <= cta_slots <= %d required", kLaneSlots);
    const uint64_t epl = events_per_launch < n_events ? events_per_launch : n_events;
    const uint64_t nl = (n_events + epl - 1) / epl;
    if (nl > kMaxLaunches) return fail(VEGAS_EINVAL, "too many launches for one iteration (raise events_per_launch)");
    int lanes = 1, grid = cta_slots, extra = 0;
    plan_launches(n_events, epl, threads_per_cta, cta_slots, &lanes, &grid, &extra);
    if (n_launches) *n_launches = static_cast<int>(nl);
    if (stream_lanes) *stream_lanes = lanes;
    if (ctas_per_launch) *ctas_per_launch = grid;
    if (extra_cta_every) *extra_cta_every = extra;
    return VEGAS_OK;
}

int vegas_partials(const vegas_ctx* c, void** dev_partials, size_t* n_doubles)
{
    if (!c) return fail(VEGAS_EINVAL, "ctx is NULL");
    if (dev_partials) *dev_partials = c->ws + c->L.part;
    if (n_doubles) *n_doubles = kPartHeader + static_cast<size_t>(c->dim) * c->nbins;
    return VEGAS_OK;
}

int vegas_finalize_enqueue(vegas_ctx* c, uint64_t n_total)
{
    if (!c) return fail(VEGAS_EINVAL, "ctx is NULL");
    if (n_total < 2) return fail(VEGAS_EINVAL, "n_events must be >= 2");
    if (!c->shard_pending) return fail(VEGAS_ESTATE, "vegas_finalize_enqueue follows vegas_iterate_shard_enqueue");
    finalize_kernel<<<1, 32, 0, c->stream>>>(reinterpret_cast<const double*>(c->ws + c->L.part), n_total,
                                             reinterpret_cast<double*>(c->ws + c->L.result));
    CUDA_TRY(cudaGetLastError());
    c->shard_pending = false;
    c->have_hist = true;
    c->have_sums = true;
    c->last_n = n_total;
    return VEGAS_OK;
}

int vegas_iterate_collect(vegas_ctx* c, double* integral, double* error, double* hist)
{
    if (!c) return fail(VEGAS_EINVAL, "ctx is NULL");
    if (!integral || !error) return fail(VEGAS_EINVAL, "integral and error are required");
    if (!c->have_sums) return fail(VEGAS_ESTATE, "no finished iteration (a shard needs vegas_finalize_enqueue first)");
    if (hist && !c->have_hist) return fail(VEGAS_ESTATE, "the histogram of the last iteration was consumed by vegas_refine");
    const size_t cells = static_cast<size_t>(c->dim) * c->nbins;
    CUDA_TRY(cudaMemcpyAsync(c->h_result, c->ws + c->L.result, 64, cudaMemcpyDeviceToHost, c->stream));
    if (hist) CUDA_TRY(cudaMemcpyAsync(c->h_result + 8, c->ws + c->L.hist, cells * 8, cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    *integral = c->h_result[0];
    *error = c->h_result[1];
    if (hist) std::memcpy(hist, c->h_result + 8, cells * 8);
    return VEGAS_OK;
}

int vegas_iterate(vegas_ctx* c, uint64_t n_events, uint64_t events_per_launch, uint64_t seed, double* integral,
                  double* error, double* hist)
{
    if (!c) return fail(VEGAS_EINVAL, "ctx is NULL");
    if (!integral || !error) return fail(VEGAS_EINVAL, "integral and error are required");
    const int rc = vegas_iterate_enqueue(c, n_events, events_per_launch, seed, nullptr);
    if (rc != VEGAS_OK) return rc;
    return vegas_iterate_collect(c, integral, error, hist);
}

int vegas_last_sums(const vegas_ctx* c, double* S1, double* S2, double* kernel_ms)
{
    if (!c) return fail(VEGAS_EINVAL, "ctx is NULL");
    if (!c->have_sums) return fail(VEGAS_ESTATE, "no iteration yet");
    CUDA_TRY(cudaMemcpyAsync(c->h_result, c->ws + c->L.result, 64, cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    if (S1) *S1 = c->h_result[2];
    if (S2) *S2 = c->h_result[3];
    if (kernel_ms) {
        if (c->last_graph) *kernel_ms = c->last_graph_ms;        // graph-replayed steps: their average device time
        else {
            if (c->n_enqueued == 0) return fail(VEGAS_ESTATE, "no iteration has been timed yet");
            float ms = 0.f;
            const int evi = static_cast<int>((c->n_enqueued - 1) % kEvPool);
            CUDA_TRY(cudaEventElapsedTime(&ms, c->evA[evi], c->evB[evi]));
            *kernel_ms = ms;
        }
    }
    return VEGAS_OK;
}

int vegas_last_npass(const vegas_ctx* c, uint64_t* npass)
{
    if (!c || !npass) return fail(VEGAS_EINVAL, "NULL argument");
    if (!c->have_sums) return fail(VEGAS_ESTATE, "no iteration yet");
    CUDA_TRY(cudaMemcpyAsync(c->h_result, c->ws + c->L.result, 64, cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    *npass = static_cast<uint64_t>(c->h_result[4]);
    return VEGAS_OK;
}

int vegas_set_histogram(vegas_ctx* c, const double* hist)
{
    if (!c || !hist) return fail(VEGAS_EINVAL, "NULL argument");
    const size_t cells = static_cast<size_t>(c->dim) * c->nbins;
    for (size_t i = 0; i < cells; ++i)
        if (!(hist[i] >= 0.0)) return fail(VEGAS_EINVAL, "histogram cell %zu is negative or NaN", i);
    CUDA_TRY(cudaMemcpyAsync(c->ws + c->L.hist, hist, cells * 8, cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));          // `hist` is pageable host memory owned by the caller
    c->have_hist = true;
    c->hist_consumed = false;
    c->shard_pending = false;
    c->accum_clean = false;
    return VEGAS_OK;
}

// Launch geometry of the refinement CTA (refine_kernel, finalize_refine_kernel): all dimensions in one CTA, as many at a
// time as fit in shared memory (at most one per warp); the steps that are independent per bin use ceil((N + 1) / 32)
// warps per dimension when the CTA has them.
static int refine_geometry(const vegas_ctx* c, int* cta_warps_out, size_t* smem_out, size_t* max_smem_out)
{
    const int N = c->nbins;
    const size_t per_dim = 4 * (static_cast<size_t>(N) + 1) * sizeof(double);
    const int warps = c->dim < 32 ? c->dim : 32;
    int cta_warps = warps * ((N + 1 + 31) / 32);
    if (cta_warps > 32) cta_warps = 32;
    const size_t max_smem = static_cast<size_t>(c->smem_optin) - kStaticSmemReserve;
    size_t smem = per_dim * static_cast<size_t>(warps);
    if (smem > max_smem) smem = (max_smem / per_dim) * per_dim;
    if (smem < per_dim) return fail(VEGAS_EINVAL, "nbins %d: one dimension's refinement does not fit in shared memory", N);
    *cta_warps_out = cta_warps; *smem_out = smem; *max_smem_out = max_smem;
    return VEGAS_OK;
}

namespace {
// S6 and S7 in one launch: the sharded step after the all-reduce (vegas_finalize_step_enqueue).  S6 is one thread's
// work on the summed partials header; it runs in the CTA's last warp, which has the fewest bins in S7's first steps.
__global__ void finalize_refine_kernel(const double* partials, unsigned long long n_events, double* result, double* edges,
                                       double* hist, int N, double alpha, double* new_edges, int d, void* table,
                                       int precision, int* status, int smem_bytes)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (threadIdx.x == blockDim.x - 1) estimate_s6(partials, n_events, result);
    refine_all(edges, hist, N, alpha, new_edges, d, table, precision, status, smem_raw, static_cast<size_t>(smem_bytes), false);
}
}  // namespace

int vegas_finalize_step_enqueue(vegas_ctx* c, uint64_t n_total, double alpha)
{
    if (!c) return fail(VEGAS_EINVAL, "ctx is NULL");
    if (n_total < 2) return fail(VEGAS_EINVAL, "n_events must be >= 2");
    if (!(alpha >= 0.0)) return fail(VEGAS_EINVAL, "alpha must be >= 0");
    if (!c->shard_pending) return fail(VEGAS_ESTATE, "vegas_finalize_step_enqueue follows vegas_iterate_shard_enqueue");
    int cta_warps = 0;
    size_t smem = 0, max_smem = 0;
    const int rc = refine_geometry(c, &cta_warps, &smem, &max_smem);
    if (rc != VEGAS_OK) return rc;
    if (smem > 48 * 1024) CUDA_TRY(cudaFuncSetAttribute(finalize_refine_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(max_smem)));
    finalize_refine_kernel<<<1, 32 * cta_warps, smem, c->stream>>>(
        reinterpret_cast<const double*>(c->ws + c->L.part), n_total, reinterpret_cast<double*>(c->ws + c->L.result),
        reinterpret_cast<double*>(c->ws + c->L.edges), reinterpret_cast<double*>(c->ws + c->L.hist), c->nbins, alpha,
        reinterpret_cast<double*>(c->ws + c->L.new_edges), c->dim, c->ws + c->L.table, c->precision == VEGAS_FP32_EVAL ? 1 : 0,
        reinterpret_cast<int*>(c->ws + c->L.status), static_cast<int>(smem));
    CUDA_TRY(cudaGetLastError());
    c->shard_pending = false;
    c->have_sums = true;
    c->last_n = n_total;
    c->have_hist = false;                                // consumed by the refinement (vegas_refine_collect hands it back
    c->hist_consumed = true;                             // if the refinement is rejected)
    c->refine_pending += 1;
    return VEGAS_OK;
}

int vegas_refine_enqueue(vegas_ctx* c, double alpha)
{
    if (!c) return fail(VEGAS_EINVAL, "ctx is NULL");
    if (!(alpha >= 0.0)) return fail(VEGAS_EINVAL, "alpha must be >= 0");
    if (!c->have_hist) return fail(VEGAS_ESTATE, "vegas_refine needs the histogram of a vegas_iterate");
    const int N = c->nbins;
    int cta_warps = 0;
    size_t smem = 0, max_smem = 0;
    const int rc = refine_geometry(c, &cta_warps, &smem, &max_smem);
    if (rc != VEGAS_OK) return rc;
    if (smem > 48 * 1024) CUDA_TRY(cudaFuncSetAttribute(refine_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(max_smem)));
    double* edges = reinterpret_cast<double*>(c->ws + c->L.edges);
    double* new_edges = reinterpret_cast<double*>(c->ws + c->L.new_edges);
    double* hist = reinterpret_cast<double*>(c->ws + c->L.hist);
    int* status = reinterpret_cast<int*>(c->ws + c->L.status);
    refine_kernel<<<1, 32 * cta_warps, smem, c->stream>>>(edges, hist, N, alpha, new_edges, c->dim, c->ws + c->L.table,
                                                      c->precision == VEGAS_FP32_EVAL ? 1 : 0, status, static_cast<int>(smem));
    CUDA_TRY(cudaGetLastError());
    c->have_hist = false;
    c->hist_consumed = true;
    c->refine_pending += 1;
    return VEGAS_OK;
}

int vegas_refine_collect(vegas_ctx* c)
{
    if (!c) return fail(VEGAS_EINVAL, "ctx is NULL");
    if (c->refine_pending == 0) return VEGAS_OK;
    int* status = reinterpret_cast<int*>(c->ws + c->L.status);
    CUDA_TRY(cudaMemcpyAsync(c->h_status, status, 3 * sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaMemsetAsync(status, 0, sizeof(int), c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    const int pending = c->refine_pending;
    c->refine_pending = 0;
    // the latest refinement was rejected and nothing overwrote H since: the histogram is still there for another try
    // (not after a fused step: its refinement clears H either way and sets no hist_consumed)
    if (c->h_status[2] != 0 && c->hist_consumed) { c->have_hist = true; c->hist_consumed = false; }
    if (c->h_status[0] != 0)
        return fail(VEGAS_EGRID, "refined edges were not strictly increasing in %d of the last %d refinement(s); each of those left its grid and histogram unchanged", c->h_status[0], pending);
    return VEGAS_OK;
}

int vegas_refine(vegas_ctx* c, double alpha)
{
    // the outcome of earlier asynchronous refinements first; a rejection among them is not dropped: it is reported
    // by this call (after this refinement was attempted) unless this call fails for a reason of its own
    const int rc0 = vegas_refine_collect(c);
    if (rc0 != VEGAS_OK && rc0 != VEGAS_EGRID) return rc0;
    int rc = vegas_refine_enqueue(c, alpha);
    if (rc != VEGAS_OK) return rc;
    rc = vegas_refine_collect(c);
    if (rc == VEGAS_OK && rc0 == VEGAS_EGRID)
        return fail(VEGAS_EGRID, "this refinement was applied, but an earlier asynchronous refinement (vegas_refine_enqueue) had been rejected: its edges were not strictly increasing and it left its grid unchanged");
    return rc;
}

int vegas_iteration_kernel_ms(const vegas_ctx* c, int back, double* kernel_ms)
{
    if (!c || !kernel_ms) return fail(VEGAS_EINVAL, "NULL argument");
    if (back < 0 || back >= kEvPool || static_cast<uint64_t>(back) >= c->n_enqueued)
        return fail(VEGAS_EINVAL, "back = %d: only the last min(%d, iterations so far) iterations keep their events", back, kEvPool);
    const int evi = static_cast<int>((c->n_enqueued - 1 - back) % kEvPool);
    CUDA_TRY(cudaEventSynchronize(c->evB[evi]));
    float ms = 0.f;
    CUDA_TRY(cudaEventElapsedTime(&ms, c->evA[evi], c->evB[evi]));
    *kernel_ms = ms;
    return VEGAS_OK;
}

int vegas_tune_events_per_launch(vegas_ctx* c, uint64_t n_events, uint64_t seed, const uint64_t* candidates,
                                 int n_candidates, uint64_t* best, double* ms)
{
    if (!c) return fail(VEGAS_EINVAL, "ctx is NULL");
    if (!candidates || !best || n_candidates < 1) return fail(VEGAS_EINVAL, "candidates, best and n_candidates >= 1 are required");
    const uint32_t it0 = c->iteration;
    int rc = VEGAS_OK;
    double best_ms = 0.0;
    for (int i = 0; i < n_candidates && rc == VEGAS_OK; ++i) {
        double t = 0.0;
        for (int rep = 0; rep < 2 && rc == VEGAS_OK; ++rep) {        // rep 0 warms up this launch geometry
            c->iteration = it0;
            rc = vegas_iterate_enqueue(c, n_events, candidates[i], seed, nullptr);
            if (rc == VEGAS_OK) rc = vegas_last_sums(c, nullptr, nullptr, &t);
        }
        if (rc != VEGAS_OK) break;
        if (ms) ms[i] = t;
        if (i == 0 || t < best_ms) { best_ms = t; *best = candidates[i]; }
    }
    c->iteration = it0;
    c->have_hist = false;
    c->have_sums = false;
    c->hist_consumed = false;
    c->shard_pending = false;
    c->accum_clean = false;
    return rc;
}

int vegas_combine_iterations(int n, const double* I, const double* sg, double* mean, double* comb_error, double* chi2_dof)
{
    if (n < 1 || !I || !sg || !mean || !comb_error) return fail(VEGAS_EINVAL, "combine: n >= 1 and non-NULL arrays/outputs required");
    double sw = 0.0, swi = 0.0, plain = 0.0;
    for (int i = 0; i < n; ++i) {
        plain += I[i];
        if (sg[i] > 0.0 && std::isfinite(sg[i]) && std::isfinite(I[i])) {
            const double w = 1.0 / (sg[i] * sg[i]);
            sw += w;
            swi += w * I[i];
        }
    }
    if (!(sw > 0.0)) {                                   // no iteration carries weight
        *mean = plain / n;
        *comb_error = 0.0;
        if (chi2_dof) *chi2_dof = 0.0;
        return VEGAS_OK;
    }
    const double m = swi / sw;
    double chi2 = 0.0;
    for (int i = 0; i < n; ++i)
        if (sg[i] > 0.0 && std::isfinite(sg[i]) && std::isfinite(I[i])) {
            const double dlt = I[i] - m;
            chi2 += dlt * dlt / (sg[i] * sg[i]);
        }
    *mean = m;
    *comb_error = 1.0 / std::sqrt(sw);
    if (chi2_dof) *chi2_dof = (n > 1) ? chi2 / (n - 1) : 0.0;
    return VEGAS_OK;
}

static void drop_step_graphs(vegas_ctx* c)
{
    if (c->gexec) { cudaGraphExecDestroy(c->gexec); c->gexec = nullptr; }
    if (c->gexec_k) { cudaGraphExecDestroy(c->gexec_k); c->gexec_k = nullptr; }
}

// Capture one whole step {memset, iterate launches, finalize, refine, commit} of (n_events, epl, seed, alpha) with
// the current launch shape into a CUDA graph (kept until the key changes).  In the captured step the iteration
// counter lives in device memory: finalize logs (I, sigma) to a ring and advances it.
static int capture_steps(vegas_ctx* c, int steps, uint64_t n_events, uint64_t epl, uint64_t seed, double alpha, cudaGraphExec_t* out)
{
    CUDA_TRY(cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeRelaxed));
    // one kernel per launch, the last CTA of the iteration refines (fused step); two kernels if the launch shape has too
    // little shared memory for that.  No memset either way: run_steps_graph_on clears the accumulators once before the
    // first replay and every step leaves them clean.
    int rc = VEGAS_OK;
    for (int k = 0; k < steps && rc == VEGAS_OK; ++k) {
        if (can_fuse_refine(c)) rc = enqueue_iteration(c, n_events, 0, n_events, epl, seed, nullptr, kGraphStep, false, alpha);
        else {
            rc = enqueue_iteration(c, n_events, 0, n_events, epl, seed, nullptr, kGraphStep, false);     // (carries its memset)
            if (rc == VEGAS_OK) { c->have_hist = true; rc = vegas_refine_enqueue(c, alpha); }
        }
    }
    cudaGraph_t graph = nullptr;
    const cudaError_t e = cudaStreamEndCapture(c->stream, &graph);     // always leave capture mode
    c->refine_pending = 0;
    if (rc != VEGAS_OK) { if (graph) cudaGraphDestroy(graph); return rc; }
    if (e != cudaSuccess) return fail(VEGAS_ECUDA, "cudaStreamEndCapture failed: %s", cudaGetErrorString(e));
    const cudaError_t e2 = cudaGraphInstantiate(out, graph, 0);
    cudaGraphDestroy(graph);
    if (e2 != cudaSuccess) { *out = nullptr; return fail(VEGAS_ECUDA, "cudaGraphInstantiate failed: %s", cudaGetErrorString(e2)); }
    return VEGAS_OK;
}

// Two graphs per key: one step, and kStepsPerGraph consecutive steps (a graph launch costs ~1 us between two steps, and
// inside one graph the kernels of consecutive single-launch steps are linked by programmatic dependent launch).
static int ensure_step_graph(vegas_ctx* c, uint64_t n_events, uint64_t epl, uint64_t seed, double alpha)
{
    if (c->gexec && c->g_n == n_events && c->g_epl == epl && c->g_seed == seed && c->g_alpha == alpha &&
        c->g_threads == c->threads && c->g_ctas == c->ctas_per_sm && c->g_rshift == c->rshift && c->g_inst == c->inst)
        return VEGAS_OK;
    drop_step_graphs(c);
    int rc = capture_steps(c, 1, n_events, epl, seed, alpha, &c->gexec);
    // many-launch steps are long enough for the graph boundary not to matter (and their graphs are large)
    if (rc == VEGAS_OK && (n_events + epl - 1) / epl == 1) rc = capture_steps(c, kStepsPerGraph, n_events, epl, seed, alpha, &c->gexec_k);
    if (rc != VEGAS_OK) { drop_step_graphs(c); return rc; }
    c->g_n = n_events; c->g_epl = epl; c->g_seed = seed; c->g_alpha = alpha;
    c->g_threads = c->threads; c->g_ctas = c->ctas_per_sm; c->g_rshift = c->rshift; c->g_inst = c->inst;
    return VEGAS_OK;
}

// `total` replays of the captured step; (I, sigma) of every iteration into I[], sg[]; average device time per
// iteration into *avg_ms.  One host synchronisation per kRing iterations.
static int run_steps_graph_on(vegas_ctx* c, int total, uint64_t n_events, uint64_t epl, uint64_t seed, double alpha,
                              double* I, double* sg, double* iter_ms);

static int run_steps_graph(vegas_ctx* c, int total, uint64_t n_events, uint64_t epl, uint64_t seed, double alpha,
                           double* I, double* sg, double* iter_ms)
{
    int rc = vegas_refine_collect(c);
    if (rc != VEGAS_OK && rc != VEGAS_EGRID) return rc;
    // fork the internal stream from the caller's, run there, join back: stream order is kept for the caller
    cudaStream_t user = c->stream;
    CUDA_TRY(cudaEventRecord(c->fork, user));
    CUDA_TRY(cudaStreamWaitEvent(c->gstream, c->fork, 0));
    c->stream = c->gstream;
    rc = run_steps_graph_on(c, total, n_events, epl, seed, alpha, I, sg, iter_ms);
    c->stream = user;
    if (cudaEventRecord(c->fork, c->gstream) == cudaSuccess) cudaStreamWaitEvent(user, c->fork, 0);
    return rc;
}

static int run_steps_graph_on(vegas_ctx* c, int total, uint64_t n_events, uint64_t epl, uint64_t seed, double alpha,
                              double* I, double* sg, double* iter_ms)
{
    int rc;
    rc = ensure_step_graph(c, n_events, epl, seed, alpha);
    if (rc != VEGAS_OK) return rc;
    uint32_t* h_it = reinterpret_cast<uint32_t*>(c->h_status) + 4;
    *h_it = c->iteration;
    CUDA_TRY(cudaMemcpyAsync(c->ws + c->L.dev_iter, h_it, 4, cudaMemcpyHostToDevice, c->stream));
    if (!c->accum_clean)                                 // the captured fused step has no memset of its own
        CUDA_TRY(cudaMemsetAsync(c->ws + c->L.zero_begin, 0, c->L.zero_end - c->L.zero_begin, c->stream));
    c->accum_clean = false;                              // until every replay below was enqueued and the run was read back
    double* ring = reinterpret_cast<double*>(c->ws + c->L.ring);
    stamp_kernel<<<1, 1, 0, c->stream>>>(ring + 3 * kRing);
    CUDA_TRY(cudaEventRecord(c->run_ev0, c->stream));
    auto stamp_of = [](double v) { long long t; std::memcpy(&t, &v, 8); return t; };
    long long t_prev = 0;
    for (int done = 0; done < total;) {
        const int chunk = (total - done < kRing) ? total - done : kRing;
        for (int i = 0; i < chunk;) {
            if (c->gexec_k && chunk - i >= kStepsPerGraph) { CUDA_TRY(cudaGraphLaunch(c->gexec_k, c->stream)); i += kStepsPerGraph; }
            else { CUDA_TRY(cudaGraphLaunch(c->gexec, c->stream)); i += 1; }
        }
        if (done + chunk == total) CUDA_TRY(cudaEventRecord(c->run_ev1, c->stream));
        CUDA_TRY(cudaMemcpyAsync(c->h_ring, ring, (kRing * 3 + 1) * 8, cudaMemcpyDeviceToHost, c->stream));
        CUDA_TRY(cudaStreamSynchronize(c->stream));
        if (done == 0) t_prev = stamp_of(c->h_ring[3 * kRing]);
        for (int i = 0; i < chunk; ++i) {
            const uint32_t it = c->iteration + static_cast<uint32_t>(done + i);
            I[done + i] = c->h_ring[3 * (it % kRing) + 0];
            sg[done + i] = c->h_ring[3 * (it % kRing) + 1];
            const long long t = stamp_of(c->h_ring[3 * (it % kRing) + 2]);
            if (iter_ms) iter_ms[done + i] = static_cast<double>(t - t_prev) * 1e-6;
            t_prev = t;
        }
        done += chunk;
    }
    float ms = 0.f;
    CUDA_TRY(cudaEventElapsedTime(&ms, c->run_ev0, c->run_ev1));
    c->last_graph = true;
    c->last_graph_ms = static_cast<double>(ms) / total;
    c->iteration += static_cast<uint32_t>(total);
    c->have_hist = false;                                // the last step refined
    c->hist_consumed = !can_fuse_refine(c);              // (a fused step clears H whatever the outcome)
    c->accum_clean = can_fuse_refine(c);
    c->have_sums = true;
    c->shard_pending = false;
    c->last_n = n_events;
    c->refine_pending = total;
    rc = vegas_refine_collect(c);
    return rc == VEGAS_EGRID ? VEGAS_OK : rc;            // a rejected refinement left its grid unchanged; the run went on
}

int vegas_set_table(vegas_ctx* c, const double* values, int n)
{
    if (!c || !values) return fail(VEGAS_EINVAL, "NULL argument");
    if (c->integrand_id != VEGAS_LO_2TO2_TAB) return fail(VEGAS_EINVAL, "this integrand takes no table");
    if (n < 4 || n > kMaxTable) return fail(VEGAS_EINVAL, "table length %d not in 4..%d", n, kMaxTable);
    CUDA_TRY(cudaMemcpyAsync(c->ws + c->L.idata, values, sizeof(double) * static_cast<size_t>(n), cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));          // `values` is pageable host memory owned by the caller
    c->ic.tab = reinterpret_cast<const double*>(c->ws + c->L.idata);
    c->ic.ntab = n;
    if (c->gexec) { cudaGraphExecDestroy(c->gexec); c->gexec = nullptr; }   // captured kernel arguments are stale
    if (c->gexec_k) { cudaGraphExecDestroy(c->gexec_k); c->gexec_k = nullptr; }
    if (c->igexec) { cudaGraphExecDestroy(c->igexec); c->igexec = nullptr; }
    return VEGAS_OK;
}

int vegas_use_cuda_graph(vegas_ctx* c, int enable)
{
    if (!c) return fail(VEGAS_EINVAL, "ctx is NULL");
    c->use_graph = enable ? 1 : 0;
    return VEGAS_OK;
}

int vegas_run_integration(vegas_ctx* c, int n_iter, int n_warmup, uint64_t n_events, uint64_t events_per_launch,
                          uint64_t seed, double alpha, double* mean, double* error, double* chi2_dof,
                          double* iter_integral, double* iter_error, double* iter_kernel_ms)
{
    if (!c) return fail(VEGAS_EINVAL, "ctx is NULL");
    if (n_iter < 1 || n_warmup < 0) return fail(VEGAS_EINVAL, "n_iter >= 1 and n_warmup >= 0 required");
    if (!mean || !error) return fail(VEGAS_EINVAL, "mean and error are required");
    const int total = n_warmup + n_iter;
    double* I = static_cast<double*>(std::malloc(sizeof(double) * 2 * static_cast<size_t>(total)));
    if (!I) return fail(VEGAS_ENOMEM, "host allocation failed");
    double* sg = I + total;
    int rc = VEGAS_OK;
    if (c->use_graph) {
        if (n_events < 2 || events_per_launch == 0) { std::free(I); return fail(VEGAS_EINVAL, "n_events >= 2 and events_per_launch > 0 required"); }
        rc = run_steps_graph(c, total, n_events, events_per_launch, seed, alpha, I, sg, iter_kernel_ms);
    } else
    for (int it = 0; it < total && rc == VEGAS_OK; ++it) {
        rc = vegas_iterate(c, n_events, events_per_launch, seed, &I[it], &sg[it], nullptr);
        if (rc != VEGAS_OK) break;
        if (iter_kernel_ms) rc = vegas_last_sums(c, nullptr, nullptr, &iter_kernel_ms[it]);
        if (rc != VEGAS_OK) break;
        rc = vegas_refine(c, alpha);
        if (rc == VEGAS_EGRID) rc = VEGAS_OK;            // grid unchanged; keep integrating
    }
    if (rc == VEGAS_OK) {
        if (iter_integral) std::memcpy(iter_integral, I, sizeof(double) * total);
        if (iter_error) std::memcpy(iter_error, sg, sizeof(double) * total);
        rc = vegas_combine_iterations(n_iter, I + n_warmup, sg + n_warmup, mean, error, chi2_dof);
    }
    std::free(I);
    return rc;
}

int vegas_get_grid(const vegas_ctx* c, double* edges)
{
    if (!c || !edges) return fail(VEGAS_EINVAL, "NULL argument");
    CUDA_TRY(cudaMemcpyAsync(edges, c->ws + c->L.edges, static_cast<size_t>(c->dim) * (c->nbins + 1) * 8, cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    return VEGAS_OK;
}

int vegas_set_grid(vegas_ctx* c, const double* edges)
{
    if (!c || !edges) return fail(VEGAS_EINVAL, "NULL argument");
    const int d = c->dim, N = c->nbins;
    for (int k = 0; k < d; ++k) {                       // argument validation (host pointer)
        const double* E = edges + static_cast<size_t>(k) * (N + 1);
        if (E[0] != 0.0 || E[N] != 1.0) return fail(VEGAS_EGRID, "dimension %d: edges must run from 0 to 1", k);
        for (int i = 0; i < N; ++i)
            if (!(E[i] < E[i + 1])) return fail(VEGAS_EGRID, "dimension %d: edges not strictly increasing at %d", k, i);
    }
    CUDA_TRY(cudaMemcpyAsync(c->ws + c->L.edges, edges, static_cast<size_t>(d) * (N + 1) * 8, cudaMemcpyHostToDevice, c->stream));
    const int rc = build_table(c, 0);
    if (rc != VEGAS_OK) return rc;
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    c->have_hist = false;                                // H was sampled through the old grid: it must not refine the new one
    c->hist_consumed = false;
    return VEGAS_OK;
}

int vegas_reset(vegas_ctx* c)
{
    if (!c) return fail(VEGAS_EINVAL, "ctx is NULL");
    const int rc = build_table(c, 1);
    if (rc != VEGAS_OK) return rc;
    CUDA_TRY(cudaMemsetAsync(c->ws + c->L.zero_begin, 0, c->L.zero_end - c->L.zero_begin, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    c->iteration = 0;
    c->have_hist = false;
    c->have_sums = false;
    c->hist_consumed = false;
    c->shard_pending = false;
    c->accum_clean = true;
    return VEGAS_OK;
}

int vegas_set_iteration(vegas_ctx* c, uint32_t iteration)
{
    if (!c) return fail(VEGAS_EINVAL, "ctx is NULL");
    c->iteration = iteration;
    return VEGAS_OK;
}

int vegas_get_iteration(const vegas_ctx* c, uint32_t* iteration)
{
    if (!c || !iteration) return fail(VEGAS_EINVAL, "NULL argument");
    *iteration = c->iteration;
    return VEGAS_OK;
}

int vegas_debug_events(vegas_ctx* c, uint64_t first_event, uint32_t count, uint64_t seed, int32_t* bins, double* x,
                       double* jac, double* f, double* wf, int32_t* pass)
{
    if (!c) return fail(VEGAS_EINVAL, "ctx is NULL");
    if (count == 0) return VEGAS_OK;
    if ((first_event & 0xFFFFFFFFull) + count > (uint64_t(1) << 32)) return fail(VEGAS_EINVAL, "range straddles a multiple of 2^32");
    // kDebugChunk events at a time through the scratch region of the caller's workspace (the library allocates no
    // device memory)
    const size_t d = static_cast<size_t>(c->dim);
    unsigned char* tmp = c->ws + c->L.scratch;
    double* d_x = reinterpret_cast<double*>(tmp);
    double* d_jac = d_x + kDebugChunk * d;
    double* d_f = d_jac + kDebugChunk;
    double* d_wf = d_f + kDebugChunk;
    int32_t* d_bins = reinterpret_cast<int32_t*>(d_wf + kDebugChunk);
    int32_t* d_pass = d_bins + kDebugChunk * d;
    for (uint32_t done = 0; done < count; done += kDebugChunk) {
        const uint32_t n = (count - done < kDebugChunk) ? count - done : kDebugChunk;
        IterArgs a;
        fill_args(c, seed, first_event + done, n, a);
        cudaError_t e = inst_debug(c->inst, a, static_cast<int>((n + 127) / 128), 128, c->stream, d_bins, d_x, d_jac, d_f, d_wf, d_pass);
        auto copy = [&](void* dst, const void* src, size_t bytes) {
            if (e == cudaSuccess && dst) e = cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, c->stream);
        };
        copy(bins ? bins + done * d : nullptr, d_bins, n * d * 4);
        copy(x ? x + done * d : nullptr, d_x, n * d * 8);
        copy(jac ? jac + done : nullptr, d_jac, static_cast<size_t>(n) * 8);
        copy(f ? f + done : nullptr, d_f, static_cast<size_t>(n) * 8);
        copy(wf ? wf + done : nullptr, d_wf, static_cast<size_t>(n) * 8);
        copy(pass ? pass + done : nullptr, d_pass, static_cast<size_t>(n) * 4);
        if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);          // the scratch region is reused by the next chunk
        if (e != cudaSuccess) return fail(VEGAS_ECUDA, "vegas_debug_events: %s", cudaGetErrorString(e));
    }
    return VEGAS_OK;
}

}  // extern "C"
