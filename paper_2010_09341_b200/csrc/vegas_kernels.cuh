// vegas_kernels.cuh -- the kernels of the Vegas hot path (sm_100a): iterate (S1-S5), finalize (S6),
// refine (S7), table staging and the per-event parity hook.  Steps and readings: DESIGN.md /
// SURVEY.md 8.c; BASELINE.json north_star names the subsystems (event generation, grid mapping,
// integrand evaluation, reduction, grid refinement, batching).  No code is shared with oracle/.
#pragma once
#include "vegas_device.cuh"

namespace vegas {

// ------------------------------------------------------------------------------------------------
// Error-free transformations for the compensated sums (S5: "Kahan-compensated in FP64").
// A compensated value is a pair (hi, lo) standing for hi + lo.
// ------------------------------------------------------------------------------------------------
struct Comp {
    double hi, lo;
};

__device__ __forceinline__ void two_sum(double a, double b, double& s, double& r)
{
    s = __dadd_rn(a, b);
    const double bb = __dsub_rn(s, a);
    r = __dadd_rn(__dsub_rn(a, __dsub_rn(s, bb)), __dsub_rn(b, bb));
}

// Kahan step: add x to (hi, lo).  lo carries the rounding error of the running sum.
__device__ __forceinline__ void kahan_add(Comp& c, double x)
{
    const double y = __dadd_rn(x, c.lo);
    const double t = __dadd_rn(c.hi, y);
    c.lo = __dsub_rn(y, __dsub_rn(t, c.hi));
    c.hi = t;
}

// (hi, lo) += (ohi, olo), exact in the leading term.
__device__ __forceinline__ void comp_add(Comp& c, double ohi, double olo)
{
    double s, r;
    two_sum(c.hi, ohi, s, r);
    c.hi = s;
    c.lo = __dadd_rn(__dadd_rn(c.lo, olo), r);
}

__device__ __forceinline__ void comp_warp_reduce(Comp& c)
{
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        const double ohi = __shfl_down_sync(0xFFFFFFFFu, c.hi, off);
        const double olo = __shfl_down_sync(0xFFFFFFFFu, c.lo, off);
        comp_add(c, ohi, olo);
    }
}

// ------------------------------------------------------------------------------------------------
// iterate_kernel: S1-S5 for the events [e_first, e_first + count) of one launch.
//
// One thread owns whole events (all d coordinates): Philox words, mantissas, bins, x, J and f stay in
// registers; the only memory traffic per event is d reads of the (lo, wd) table and d fp64 updates of
// the histogram, both in shared memory.  HBM: one table read per CTA at entry, one d*N flush per CTA
// at exit (global fp64 reductions), four doubles per CTA for the scalar sums.
//
// Shared memory:  hist[d*N][R] fp64 | table[d*N][TREP] real2 | per-warp partial sums.
//   hist : R = 2^rshift lane-indexed replicas; lane l updates replica l%R, so with R = 32 no two lanes of a
//          warp ever touch the same word and the compare-and-swap that an fp64 shared-memory add is on
//          sm_100a (LDS, DADD, ATOMS.CAST) succeeds first try unless another warp got in between.
//   table: TREP lane-indexed copies of every 16-byte (fp64) / 8-byte (fp32) cell, lane l reads copy
//          l%TREP.  A 16-byte shared load is served one quarter-warp (8 lanes) per wavefront; with TREP = 8
//          the 8 lanes hit 8 different 4-bank groups whatever their bins are, so the random-bin lookup
//          costs 3.0 wavefronts per load (profiles/r03_ncu_full_cfg2_iterate.md) instead of the ~9.6 measured in round 1 without replication.
// Template parameters: D, NB compile-time dimension / bin count (0 = run-time a.dim / a.nbins); RS
// compile-time log2 R (-1 = run-time a.rshift); TREP; HB = number of histogram updates whose
// compare-and-swap sequences are issued together (0 = one atomicAdd spin loop per update).
// Grid: a multiple of the SM count; the events of the launch are dealt round-robin to threads
// (idx = blockIdx*blockDim + tid, stride gridDim*blockDim), so the Philox counter of a thread's next
// event is its previous one plus a constant.
// ------------------------------------------------------------------------------------------------
constexpr int kQueueCap = 64;   // entries of the per-warp compaction ring buffer (power of two >= 64)

template <int D>
struct BinPack {   // d bin indices, 16 bits each, kept in registers (all indices are compile-time)
    uint32_t w[((D ? D : kMaxDim) + 1) / 2];
    __device__ __forceinline__ void clear()
    {
#pragma unroll
        for (int i = 0; i < ((D ? D : kMaxDim) + 1) / 2; ++i) w[i] = 0u;
    }
    __device__ __forceinline__ void set(int k, int i) { w[k >> 1] |= static_cast<uint32_t>(i) << ((k & 1) * 16); }
    __device__ __forceinline__ int get(int k) const { return static_cast<int>((w[k >> 1] >> ((k & 1) * 16)) & 0xFFFFu); }
};

// fp64 histogram cells in shared memory, addressed by 32-bit shared-window address.  On sm_100a an fp64 add on shared
// memory is a compare-and-swap loop (LDS.64, DADD, ATOMS.CAS.64); written out here so that several chains can be
// issued together and the lost-race test of a whole batch is one predicate.
__device__ __forceinline__ unsigned long long hist_load(uint32_t addr)
{
    unsigned long long v;
    asm volatile("ld.shared.u64 %0, [%1];" : "=l"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ unsigned long long hist_cas(uint32_t addr, unsigned long long expect, unsigned long long desired)
{
    unsigned long long old;
    asm volatile("atom.shared.cas.b64 %0, [%1], %2, %3;" : "=l"(old) : "r"(addr), "l"(expect), "l"(desired) : "memory");
    return old;
}
__device__ __forceinline__ unsigned long long add_bits(unsigned long long bits, double q)
{
    return static_cast<unsigned long long>(__double_as_longlong(__dadd_rn(__longlong_as_double(static_cast<long long>(bits)), q)));
}
// A lost race: one more swap from the value the failed one returned (no reload: the window in which yet another warp
// can get in between is a DADD long, and on the headline workload this second attempt practically always succeeds);
// if that is lost too the word is contended and the update falls back to atomicAdd, which on an fp64 word in shared
// memory is the loop LDS.64, DADD, ATOMS.CAST.SPIN.64, branch.  Measured: looping on plain
// ATOMS.CAS.64 with the returned value instead is much worse whenever several lanes or warps really collide -- cfg1
// (all warps of a CTA reach the histogram together) +40 % shared-atomic wavefronts and +5 us per launch, cfg4 (R = 8:
// four lanes of a warp share a replica) 4.2 -> 7.7-8.3 ms; going to atomicAdd straight away costs cfg2 3 %.
__device__ __forceinline__ void hist_retry(uint32_t addr, unsigned long long seen, double q)
{
    const unsigned long long again = hist_cas(addr, seen, add_bits(seen, q));
    if (again != seen) atomicAdd(static_cast<double*>(__cvta_shared_to_generic(addr)), q);
}

// H[k][bin_k] += q for the dims [k0, k0 + HB): all loads, then all adds, then all compare-and-swaps, so the HB
// dependent chains (LDS -> DADD -> ATOMS.CAS) overlap; the differences (returned ^ expected) are OR-ed into one
// word (two three-input logic ops per update, opaque to the compiler so that it does not turn them into a
// predicate per update) and tested once; a lost race (another warp updated the same replica word in between -- rare
// with lane-indexed replicas) is redone by hist_retry.  `hist_lane` = shared address of this lane's replica of
// cell 0; cells are HCELL bytes apart (0: run-time, 8 << rs).
__device__ __forceinline__ uint32_t or_xor(uint32_t acc, uint32_t a, uint32_t b)
{
    uint32_t v = acc | (a ^ b);                          // one three-input logic op
    asm("" : "+r"(v));                                   // opaque: keeps it a data value instead of a predicate chain
    return v;
}

template <int D, int NB, int HCELL, int HB>
__device__ __forceinline__ void hist_update_batch(uint32_t hist_lane, int k0, int d, uint32_t N, int rs, const BinPack<D>& bp,
                                                  double q)
{
    uint32_t p[HB], off[HB];
    unsigned long long o[HB], r[HB];
    uint32_t diff = 0u;
#pragma unroll
    for (int j = 0; j < HB; ++j) {
        const int k = k0 + j;
        if (k < d) {
            if constexpr (HCELL > 0) {
                p[j] = hist_lane + static_cast<uint32_t>(bp.get(k)) * HCELL;
                off[j] = static_cast<uint32_t>(k) * N * HCELL;       // an immediate when D and NB are compile-time
            } else {
                p[j] = hist_lane + ((static_cast<uint32_t>(k) * N + static_cast<uint32_t>(bp.get(k))) << (3 + rs));
                off[j] = 0u;
            }
            o[j] = hist_load(p[j] + off[j]);
        }
    }
#pragma unroll
    for (int j = 0; j < HB; ++j)
        if (k0 + j < d) {
            r[j] = hist_cas(p[j] + off[j], o[j], add_bits(o[j], q));
            diff = or_xor(diff, static_cast<uint32_t>(r[j]), static_cast<uint32_t>(o[j]));
            diff = or_xor(diff, static_cast<uint32_t>(r[j] >> 32), static_cast<uint32_t>(o[j] >> 32));
        }
    if (diff != 0u) {
#pragma unroll
        for (int j = 0; j < HB; ++j)
            if (k0 + j < d && r[j] != o[j]) hist_retry(p[j] + off[j], r[j], q);
    }
}

// one update with the plain spin loop (HB == 0): atomicAdd on an fp64 word in shared memory compiles to the tight loop
// LDS.64, DADD, ATOMS.CAST.SPIN.64 (swap + success predicate in one instruction), branch -- the form to use when lost
// races are frequent (few replicas: lanes of one warp that share a replica and a bin collide)
__device__ __forceinline__ void hist_update_one(double* cell, double q)
{
    atomicAdd(cell, q);
}

__device__ __forceinline__ void finalize_warp(const double* slots, int nlanes, int lane_stride, int per_lane,
                                              const unsigned long long* npass, unsigned long long n_events,
                                              double* partials, double* result, uint32_t* dev_iter, double* ring,
                                              int ring_len);

__device__ __forceinline__ void refine_all(double* edges, double* hist, int N, double alpha, double* new_edges, int d,
                                           void* table, int precision, int* status, unsigned char* smem, size_t smem_bytes,
                                           bool clear_hist_always);

// What every CTA of an iterate launch does after its events: the CTA's compensated sums go to its slot, the replicas of
// its `cells` histogram cells (global cells cell0 ...) are summed and reduced into H, and the CTA that finishes last
// over all launches of the iteration runs S6 -- and, in a fused step, S7.
__device__ __forceinline__ void cta_tail(const IterArgs& a, Comp s1, Comp s2, unsigned int np, const double* sh_hist,
                                         double* sh_part, int cells, int cell0, int rs, int d, int N, unsigned char* smem_raw)
{
    const int tid = threadIdx.x, lane = tid & 31;
    const int R = 1 << rs;
    // ---- scalar sums: warp shuffle tree on compensated pairs, then one thread per CTA ----
    comp_warp_reduce(s1);
    comp_warp_reduce(s2);
    np = __reduce_add_sync(0xFFFFFFFFu, np);
    const int warp = tid >> 5, nwarps = (blockDim.x + 31) >> 5;
    if (lane == 0) {
        sh_part[warp * 5 + 0] = s1.hi; sh_part[warp * 5 + 1] = s1.lo;
        sh_part[warp * 5 + 2] = s2.hi; sh_part[warp * 5 + 3] = s2.lo;
        sh_part[warp * 5 + 4] = static_cast<double>(np);
    }
    __syncthreads();
    if (warp == 0) {
        // the warps' partial sums (at most 32) go through the same compensated shuffle tree, then into the CTA's slot,
        // which carries over from the previous launches of this iteration (stream order)
        Comp t1{0.0, 0.0}, t2{0.0, 0.0};
        unsigned int npw = 0u;
        if (lane < nwarps) {
            t1.hi = sh_part[lane * 5 + 0]; t1.lo = sh_part[lane * 5 + 1];
            t2.hi = sh_part[lane * 5 + 2]; t2.lo = sh_part[lane * 5 + 3];
            npw = static_cast<unsigned int>(sh_part[lane * 5 + 4]);
        }
        comp_warp_reduce(t1);
        comp_warp_reduce(t2);
        const unsigned int npb = __reduce_add_sync(0xFFFFFFFFu, npw);     // <= 32 * 2^26 events of one launch per CTA: no overflow
        if (lane == 0) {
            double* slot = a.slots + static_cast<size_t>(blockIdx.x) * 4;
            comp_add(t1, slot[0], slot[1]);
            comp_add(t2, slot[2], slot[3]);
            slot[0] = t1.hi; slot[1] = t1.lo; slot[2] = t2.hi; slot[3] = t2.lo;
            if (npb) atomicAdd(a.npass, static_cast<unsigned long long>(npb));
        }
    }

    // ---- histogram flush: fixed-order sum over the replicas, one global reduction per touched cell ----
    for (int c = tid; c < cells; c += blockDim.x) {
        const double* p = sh_hist + (static_cast<size_t>(c) << rs);
        double v = p[c & (R - 1)];                              // rotated start: conflict-free reads
        for (int r = 1; r < R; ++r) v = __dadd_rn(v, p[(r + c) & (R - 1)]);
        if (v != 0.0) atomicAdd(a.hist + cell0 + c, v);
    }

    // ---- S6 in the CTA that finishes last over all launches of this iteration ----
    __shared__ int sh_last;
    __syncthreads();                                     // this CTA's slot is written
    if (tid == 0) {
        __threadfence();
        sh_last = (atomicAdd(a.ticket, 1u) == a.total_ctas - 1u);
    }
    __syncthreads();
    if (!sh_last) return;
    __threadfence();                                     // see the other CTAs' slots and histogram reductions
    // S6 by one warp.  In a fused step it is the CTA's last warp, which has the least to do in the first steps of S7
    // (no bins of its own to load), so that S6 runs beside them; S7's block barriers then order S6's reads of the slots
    // and the pass counter before they are cleared below.
    const bool fused = a.refine_alpha >= 0.0;
    if (warp == (fused ? nwarps - 1 : 0))
        finalize_warp(a.slots0, a.fin_lanes, a.fin_stride, a.fin_used, a.npass, a.n_events, a.partials, a.result,
                      a.dev_iter, a.ring, a.ring_len);
    if (fused) {
        // ---- fused step: S7 by the same CTA, in the shared memory the event loop no longer needs; then the
        // accumulators are cleared, so the next step needs no memset ----
        refine_all(a.edges, a.hist, N, a.refine_alpha, a.new_edges, d, const_cast<void*>(a.table), a.precision, a.status,
                   smem_raw, static_cast<size_t>(a.smem_bytes), true);
        for (int i = tid; i < a.fin_lanes * a.fin_used * 4; i += blockDim.x) a.slots0[i] = 0.0;
        if (tid == 0) { *a.npass = 0ull; *a.ticket = 0u; }
    }
}

template <class F, int D, int NB, int RS, int TREP, int HB, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB) iterate_kernel(const __grid_constant__ IterArgs a)
{
    using real = typename F::real;
    using real2 = typename std::conditional<sizeof(real) == 8, double2, float2>::type;
    extern __shared__ __align__(16) unsigned char smem_raw[];

    const int d = D ? D : a.dim;
    const int N = NB ? NB : a.nbins;
    const int rs = (RS >= 0) ? RS : a.rshift;
    const int cells = d * N;
    const int R = 1 << rs;
    const size_t hist_bytes = (static_cast<size_t>(cells) * R * sizeof(double) + 15) & ~size_t(15);
    const size_t tab_bytes = (static_cast<size_t>(cells) * TREP * sizeof(real2) + 15) & ~size_t(15);
    double* sh_hist = reinterpret_cast<double*>(smem_raw);
    real2* sh_tab = reinterpret_cast<real2*>(smem_raw + hist_bytes);
    double* sh_part = reinterpret_cast<double*>(smem_raw + hist_bytes + tab_bytes);

    const int tid = threadIdx.x;
    const int lane = tid & 31;
    // Programmatic dependent launch: the launch that follows this one on the stream may start now and run its own
    // prologue up to its griddepcontrol.wait, which returns once this whole grid has completed and its writes are
    // visible.  Everything before the wait touches shared memory only; the table (rewritten by the previous step's
    // refinement), the iteration counter, the slots and H are read or written after it.  Without the launch attribute
    // (or with no kernel in front) both instructions do nothing.
    asm volatile("griddepcontrol.launch_dependents;");
    for (int i = tid; i < cells * R; i += blockDim.x) sh_hist[i] = 0.0;
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const uint32_t it = a.iter_ptr ? *a.iter_ptr : a.iteration;   // S1 counter word 2
    {
        const real2* gt = static_cast<const real2*>(a.table);
        for (int i = tid; i < cells * TREP; i += blockDim.x) sh_tab[i] = gt[i / TREP];
    }
    __syncthreads();
    // lds_cell reads the staged table through plain (non-volatile, no clobber) inline asm, which the compiler sees as a
    // pure function of the address: this compiler-level fence is what keeps those reads behind the stores above and
    // the barrier (no instruction is emitted)
    asm volatile("" ::: "memory");

    constexpr int kTCell = TREP * static_cast<int>(sizeof(real2));       // bytes between the table copies of two cells
    constexpr int kHCell = (RS >= 0) ? (8 << (RS >= 0 ? RS : 0)) : 0;    // bytes between two cells' replicas (0: run-time)
    const uint32_t hist_lane = smem_addr(sh_hist) + static_cast<uint32_t>(lane & (R - 1)) * 8u;
    const uint32_t tab_lane = smem_addr(sh_tab) + static_cast<uint32_t>(lane & (TREP - 1)) * static_cast<uint32_t>(sizeof(real2));
    Comp s1{0.0, 0.0}, s2{0.0, 0.0};
    unsigned int np = 0;
    const uint32_t stride = gridDim.x * blockDim.x;

    // S4 + S5 for one event whose integrand value is known
    auto accumulate = [&](real J, real f, const BinPack<D>& bp) {
        const double wf = __dmul_rn(static_cast<double>(J), static_cast<double>(f));   // S4
        const double q = __dmul_rn(wf, wf);
        kahan_add(s1, wf);                                        // S5
        kahan_add(s2, q);
        if constexpr (HB > 0) {
#pragma unroll
            for (int k0 = 0; k0 < (D ? D : kMaxDim); k0 += HB) {
                if (!D && k0 >= d) break;
                hist_update_batch<D, NB, kHCell, HB>(hist_lane, k0, d, static_cast<uint32_t>(N), rs, bp, q);
            }
        } else {
#pragma unroll
            for (int k = 0; k < (D ? D : kMaxDim); ++k) {
                if (!D && k >= d) break;
                hist_update_one(sh_hist + (static_cast<size_t>(k * N + bp.get(k)) << rs) + (lane & (R - 1)), q);
            }
        }
    };

    if constexpr (!F::kHasCut) {
        for (uint32_t idx = blockIdx.x * blockDim.x + tid; idx < a.count; idx += stride) {
            BinPack<D> bp;
            bp.clear();
            F integrand;
            const real J = event_front<F, D, NB, kTCell>(a, it, a.e_lo_first + idx, nullptr, tab_lane,
                                                         [&](int k, int i, real) { bp.set(k, i); }, integrand);
            accumulate(J, integrand.end(a.ic, d), bp);
            np += 1u;
        }
    } else {
        // Integrands with cuts (lo_2to2 rejects ~55 % of the events): warp-level compaction.  Every lane
        // draws and maps an event and tests the cuts (cheap); events that pass are pushed to a per-warp
        // ring buffer in shared memory (ballot + popc prefix), and whenever 32 are queued the warp pops
        // them and evaluates the matrix element, weight and histogram updates with all lanes busy.
        // Rejected events contribute wf = 0 (adding 0 is the identity, reading R8).
        constexpr int QF = static_cast<int>(sizeof(F) / sizeof(double));      // integrand state
        constexpr int QB = (static_cast<int>(sizeof(BinPack<D>) / 4) + 1) / 2;  // packed bins, 8-byte words
        constexpr int QE = QF + 1 + QB;
        static_assert(sizeof(F) % sizeof(double) == 0 && sizeof(real) == 8, "queue layout assumes fp64 integrand state");
        double* queue = sh_part + ((blockDim.x + 31) >> 5) * 5 + static_cast<size_t>(tid >> 5) * (QE * kQueueCap);
        int head = 0, qn = 0;
        auto consume = [&](int pos) {
            F integrand;
            double* st = reinterpret_cast<double*>(&integrand);
#pragma unroll
            for (int j = 0; j < QF; ++j) st[j] = queue[j * kQueueCap + pos];
            const double J = queue[QF * kQueueCap + pos];
            BinPack<D> bp;
#pragma unroll
            for (int j = 0; j < QB; ++j) {
                const long long v = __double_as_longlong(queue[(QF + 1 + j) * kQueueCap + pos]);
                bp.w[2 * j] = static_cast<uint32_t>(v);
                if (2 * j + 1 < static_cast<int>(sizeof(BinPack<D>) / 4)) bp.w[2 * j + 1] = static_cast<uint32_t>(v >> 32);
            }
            accumulate(J, integrand.end(a.ic, d), bp);
        };
        for (uint32_t base = blockIdx.x * blockDim.x + (tid & ~31); base < a.count; base += stride) {
            const uint32_t idx = base + lane;
            bool pass = false;
            F integrand;
            BinPack<D> bp;
            real J = real(0);
            if (idx < a.count) {
                bp.clear();
                J = event_front<F, D, NB, kTCell>(a, it, a.e_lo_first + idx, nullptr, tab_lane,
                                                  [&](int k, int i, real) { bp.set(k, i); }, integrand);
                pass = integrand.precheck(a.ic);
            }
            const unsigned m = __ballot_sync(0xFFFFFFFFu, pass);
            if (pass) {
                const int pos = (head + qn + __popc(m & ((1u << lane) - 1u))) & (kQueueCap - 1);
                const double* st = reinterpret_cast<const double*>(&integrand);
#pragma unroll
                for (int j = 0; j < QF; ++j) queue[j * kQueueCap + pos] = st[j];
                queue[QF * kQueueCap + pos] = J;
#pragma unroll
                for (int j = 0; j < QB; ++j) {
                    unsigned long long v = bp.w[2 * j];
                    if (2 * j + 1 < static_cast<int>(sizeof(BinPack<D>) / 4)) v |= static_cast<unsigned long long>(bp.w[2 * j + 1]) << 32;
                    queue[(QF + 1 + j) * kQueueCap + pos] = __longlong_as_double(static_cast<long long>(v));
                }
            }
            qn += __popc(m);
            np += pass ? 1u : 0u;
            __syncwarp();
            if (qn >= 32) {
                consume((head + lane) & (kQueueCap - 1));
                head = (head + 32) & (kQueueCap - 1);
                qn -= 32;
                __syncwarp();
            }
        }
        if (lane < qn) consume((head + lane) & (kQueueCap - 1));
    }

    cta_tail(a, s1, s2, np, sh_hist, sh_part, cells, 0, rs, d, N, smem_raw);
}

// ------------------------------------------------------------------------------------------------
// finalize_warp, run by the first warp of the CTA that finishes last: fixed-order compensated sum of the
// per-CTA slots into the partials header
//   partials[0..4] = S1.hi, S1.lo, S2.hi, S2.lo, npass        (H follows the 8-double header in memory)
// and then, unless this launch is a shard of an iteration that other GPUs share (n_events == 0: the sums are
// all-reduced first and S6 runs in finalize_kernel), S6:
//   I = S1/n ; V = (S2/n - I*I)/(n-1) ; sigma = sqrt(max(V, 0)).
// One warp; lane l folds slots l, l+32, ... (over the per-stream-lane regions) then a shuffle tree: the order
// depends only on the launch geometry.
// result[0..5] = I, sigma, S1, S2, npass, n
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned long long global_timer_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

__device__ __forceinline__ void estimate_s6(const double* partials, unsigned long long n_events, double* result)
{
    const double S1 = __dadd_rn(partials[0], partials[1]), S2 = __dadd_rn(partials[2], partials[3]);
    const double n = static_cast<double>(n_events);
    const double I = __ddiv_rn(S1, n);
    const double V = __ddiv_rn(__dsub_rn(__ddiv_rn(S2, n), __dmul_rn(I, I)), __dsub_rn(n, 1.0));
    result[0] = I;
    result[1] = sqrt(V > 0.0 ? V : 0.0);
    result[2] = S1;
    result[3] = S2;
    result[4] = partials[4];
    result[5] = n;
}

__device__ __forceinline__ void finalize_warp(const double* slots, int nlanes, int lane_stride, int per_lane,
                                              const unsigned long long* npass, unsigned long long n_events,
                                              double* partials, double* result, uint32_t* dev_iter, double* ring,
                                              int ring_len)
{
    const int lane = threadIdx.x & 31;
    Comp t1{0.0, 0.0}, t2{0.0, 0.0};
    for (int e = lane; e < nlanes * per_lane; e += 32) {         // slot region of stream-lane e / per_lane
        const size_t s = static_cast<size_t>(e / per_lane) * lane_stride + (e % per_lane);
        comp_add(t1, __ldcg(slots + s * 4 + 0), __ldcg(slots + s * 4 + 1));   // written by other CTAs: L2 reads
        comp_add(t2, __ldcg(slots + s * 4 + 2), __ldcg(slots + s * 4 + 3));
    }
    comp_warp_reduce(t1);
    comp_warp_reduce(t2);
    if (lane == 0) {
        // renormalise the pairs so that |lo| <= ulp(hi)/2.  Across G GPUs the all-reduce adds the hi parts and the lo
        // parts separately in plain fp64: the lo parts keep each GPU's own compensation, but the G - 1 additions of hi
        // parts round, so the multi-GPU sum is within (G - 1) ulp/2 of the exact one (1e-15 relative at G = 8), not
        // compensated like the single-GPU sum
        double h1, l1, h2, l2;
        two_sum(t1.hi, t1.lo, h1, l1);
        two_sum(t2.hi, t2.lo, h2, l2);
        partials[0] = h1; partials[1] = l1; partials[2] = h2; partials[3] = l2;
        partials[4] = static_cast<double>(__ldcg(npass));
        if (n_events == 0ull) return;                    // shard: S6 after the all-reduce (finalize_kernel)
        estimate_s6(partials, n_events, result);
        if (ring) {                                      // graph replays: log (I, sigma) and advance the counter
            const uint32_t it = *dev_iter;
            ring[3 * (it % ring_len) + 0] = result[0];
            ring[3 * (it % ring_len) + 1] = result[1];
            ring[3 * (it % ring_len) + 2] = __longlong_as_double(static_cast<long long>(global_timer_ns()));   // log_time
            *dev_iter = it + 1u;
        }
    }
}

// Time stamp (ns, %globaltimer) written at the start of a graph-replayed run: the first iteration's device time is
// measured from it, every later one from the previous iteration's S6 (PAPER.md:L79 log_time).
__global__ void stamp_kernel(double* slot) { *slot = __longlong_as_double(static_cast<long long>(global_timer_ns())); }

// S6 from the partials header after the sums of all shards were added (NEXT-2: one all-reduce per iteration of
// {S1.hi, S1.lo, S2.hi, S2.lo, npass, pad[3], H[d*N]}).  One thread.
__global__ void finalize_kernel(const double* __restrict__ partials, unsigned long long n_events, double* __restrict__ result)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) estimate_s6(partials, n_events, result);
}

// ------------------------------------------------------------------------------------------------
// Grid state kernels.  Master edges E[d][N+1] are fp64; the mapping table holds (lo, wd) per cell in the
// working precision (S2):  uniform grid: lo = rnd(E[i]), wd = rnd(fl64(1/N));
//                          otherwise:    lo = rnd(E[i]), wd = rnd(fl64(E[i+1]-E[i])).
// g = fl(N*wd) is recomputed per event from wd (one multiply; same bits as a stored g).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void write_table_cell(void* table, int precision, size_t cell, double lo, double wd)
{
    if (precision == 0) static_cast<double2*>(table)[cell] = make_double2(lo, wd);
    else static_cast<float2*>(table)[cell] = make_float2(__double2float_rn(lo), __double2float_rn(wd));
}

// one CTA per dimension.  uniform != 0: also (re)writes E[k][i] = fl64(i/N), E[k][N] = 1.
__global__ void build_table_kernel(double* __restrict__ edges, void* __restrict__ table, int N, int precision,
                                   int uniform)
{
    const int k = blockIdx.x;
    double* E = edges + static_cast<size_t>(k) * (N + 1);
    if (uniform) {
        const double Nd = static_cast<double>(N);
        for (int i = threadIdx.x; i <= N; i += blockDim.x) E[i] = (i == N) ? 1.0 : __ddiv_rn(static_cast<double>(i), Nd);
        __syncthreads();
        const double wd = __ddiv_rn(1.0, Nd);
        for (int i = threadIdx.x; i < N; i += blockDim.x)
            write_table_cell(table, precision, static_cast<size_t>(k) * N + i, E[i], wd);
    } else {
        for (int i = threadIdx.x; i < N; i += blockDim.x)
            write_table_cell(table, precision, static_cast<size_t>(k) * N + i, E[i], __dsub_rn(E[i + 1], E[i]));
    }
}

// S7 (refine): all dimensions in ONE CTA, so that the all-or-nothing commit of step 7 needs
// no grid-wide dependency.  The refinement is latency-bound (d*N <= a few thousand cells, chains of dependent fp64
// operations at ~40 cycles each), so everything that the definition states as a sequential sum is done as a
// lane-chunked sum / scan instead: lane l owns the contiguous bins [l*chunk, (l+1)*chunk), sums or scans them locally
// and the 32 chunk totals are combined with shuffles (reading R12' in DESIGN.md: the summation ORDER of steps 1, 3 and 5
// is not the definition's, which moves the sums by a few ulp and the edges by ~1e-16, against a tolerance of 1e-12).
// Step 6's "smallest i with c_{i+1} >= t and m_i > 0" is a binary search over the non-decreasing prefix sums (the
// smallest i with c_{i+1} >= t has c_i < t <= c_{i+1}, hence m_i > 0: the same bin the linear scan finds; N-1 if none).
// Per-dimension shared memory: A[N+1] (h, then m) | B[N+1] (s, then the new edges) | cum[N+1] | E[N+1].
__device__ __forceinline__ double warp_sum_all(double v)
{
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v = __dadd_rn(v, __shfl_xor_sync(0xFFFFFFFFu, v, off));
    return v;                                            // identical in every lane
}

// m = x^alpha for the damping of step 4; the exponents the configurations use avoid the ~150 dependent fp64
// operations of pow() (values within 1 ulp of it)
__device__ __forceinline__ double damp_pow(double x, double alpha)
{
    if (alpha == 1.5) return __dmul_rn(x, sqrt(x));
    if (alpha == 1.0) return x;
    if (alpha == 0.5) return sqrt(x);
    if (alpha == 2.0) return __dmul_rn(x, x);
    return pow(x, alpha);
}

// The warp-level pieces of S7 for one dimension (called by the warp that owns the dimension; lane l owns the
// contiguous bins [lo, hi)).  Each returns its result in every lane.
__device__ __forceinline__ double refine_chunk_sum(const double* v, int lo, int hi)
{
    double part = 0.0;
    for (int i = lo; i < hi; ++i) part = __dadd_rn(part, v[i]);
    return warp_sum_all(part);
}

// steps 5: prefix sums cum[1..N] of m[0..N-1] (chunk-local prefix, scan of the 32 chunk totals, exact max-scan so that
// the prefix sums never decrease across a chunk boundary), cum[0] = 0.  Returns cum[N].
__device__ __forceinline__ double refine_prefix(const double* m, double* cum, int N, int lo, int hi)
{
    const int lane = threadIdx.x & 31;
    double part = 0.0;
    for (int i = lo; i < hi; ++i) {
        part = __dadd_rn(part, m[i]);
        cum[i + 1] = part;                               // chunk-local for now
    }
    double incl = part;                                  // inclusive scan of the 32 chunk totals
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const double o = __shfl_up_sync(0xFFFFFFFFu, incl, off);
        if (lane >= off) incl = __dadd_rn(incl, o);
    }
    double offset = __shfl_up_sync(0xFFFFFFFFu, incl, 1);
    if (lane == 0) offset = 0.0;
    // The prefix sums must not decrease across a chunk boundary (its two sides are rounded along different paths, so
    // they can be out of order by an ulp): every chunk is clamped from below by the largest value any earlier chunk
    // ends with -- a max-scan, which is exact.  Within a chunk fl(offset + local prefix) is non-decreasing already.
    double endmax = (hi > lo) ? __dadd_rn(offset, part) : 0.0;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const double o = __shfl_up_sync(0xFFFFFFFFu, endmax, off);
        if (lane >= off && o > endmax) endmax = o;
    }
    double floor_ = __shfl_up_sync(0xFFFFFFFFu, endmax, 1);
    if (lane == 0) floor_ = 0.0;
    for (int i = lo; i < hi; ++i) {
        const double v = __dadd_rn(offset, cum[i + 1]);
        cum[i + 1] = v > floor_ ? v : floor_;
    }
    if (lane == 0) cum[0] = 0.0;
    __syncwarp();
    return cum[N];
}

// All of S7 by one CTA, in passes of as many dimensions as fit in `smem_bytes` of shared memory (at most one per warp).
// The sums and scans of a dimension are done by ONE warp (lane-chunked, so that their order depends on N only); the
// steps that are independent per bin or per edge -- smoothing (2), damping (4: a division, a logarithm, a division and
// a power per bin), the search and interpolation of the new edges (6) and the check (7) -- are spread over all the
// warps the CTA has per dimension (cfg1 in the fused step: 8 warps for 50 bins), with a block barrier between the
// steps: the refinement is a chain of dependent fp64 operations at ~40 cycles each, and this shortens the chain.
// Then step 7 for all dimensions: if every one passed, the candidate edges become the master edges, the table is
// rebuilt and H is cleared; otherwise nothing changes (H included, so the caller may refine again, e.g. with another
// alpha) and status[0] counts the rejection (the host clears it when it collects the outcome of the refinements
// enqueued since); status[2] = the latest outcome.
__device__ __forceinline__ void refine_all(double* edges, double* hist, int N, double alpha, double* new_edges, int d,
                                           void* table, int precision, int* status, unsigned char* smem, size_t smem_bytes,
                                           bool clear_hist_always)
{
    __shared__ int sh_bad;
    __shared__ int sh_skip[kMaxDim];                     // the dimension has nothing to adapt to: edges unchanged
    __shared__ double sh_ssum[kMaxDim], sh_delta[kMaxDim];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarps = blockDim.x >> 5;
    const size_t per_dim = 4 * (static_cast<size_t>(N) + 1);            // doubles
    int group = static_cast<int>(smem_bytes / (per_dim * sizeof(double)));
    if (group > nwarps) group = nwarps;
    if (group > kMaxDim) group = kMaxDim;
    const int chunk = (N + 31) >> 5;
    const int lo = lane * chunk < N ? lane * chunk : N, hi = (lo + chunk < N) ? lo + chunk : N;
    if (tid == 0) sh_bad = 0;                            // first set after several block barriers (step 7 check)
    for (int k0 = 0; k0 < d; k0 += group) {
        const int nd = (d - k0 < group) ? d - k0 : group;
        const int wpd = nwarps / nd;                     // warps per dimension in the element-wise steps (>= 1)
        const int kk = warp / wpd;                       // this thread's dimension in those steps (>= nd: idle)
        const int e0 = (warp - kk * wpd) * 32 + lane, estride = wpd * 32;
        double* sm = reinterpret_cast<double*>(smem);
        double* A = sm + static_cast<size_t>(kk < nd ? kk : 0) * per_dim;   // [N+1] h, then m
        double* B = A + (N + 1);                         // [N+1] s, then the new edges
        double* cum = B + (N + 1);                       // [N+1]
        double* E = cum + (N + 1);                       // [N+1]
        const bool active = kk < nd;
        const int k = k0 + kk;
        // the sums and scans of dimension kk belong to the LAST warp of its group, which has the fewest (mostly no) bins
        // in the element-wise steps
        const int own = (active && warp - kk * wpd == wpd - 1) ? kk : -1;
        if (active) {                                    // H was reduced into L2 by other CTAs
            for (int i = e0; i < N; i += estride) A[i] = __ldcg(hist + static_cast<size_t>(k) * N + i);
            for (int i = e0; i <= N; i += estride) E[i] = __ldcg(edges + static_cast<size_t>(k) * (N + 1) + i);
        }
        __syncthreads();
        if (own >= 0) {                                  // step 1, by the warp that owns the dimension
            const double tot = refine_chunk_sum(A, lo, hi);
            if (lane == 0) sh_skip[own] = (!(tot > 0.0) || !isfinite(tot)) ? 1 : 0;
        }
        if (active)                                      // step 2 at the same time: it does not depend on the total
            for (int i = e0; i < N; i += estride) {
                double v;
                if (i == 0) v = __ddiv_rn(__dadd_rn(A[0], A[1]), 2.0);
                else if (i == N - 1) v = __ddiv_rn(__dadd_rn(A[N - 2], A[N - 1]), 2.0);
                else v = __ddiv_rn(__dadd_rn(__dadd_rn(A[i - 1], A[i]), A[i + 1]), 3.0);
                B[i] = v;
            }
        __syncthreads();
        const bool skip = active && sh_skip[kk] != 0;
        if (own >= 0 && !skip) {                         // step 3
            const double ssum = refine_chunk_sum(B, lo, hi);
            if (lane == 0) sh_ssum[own] = ssum;
        }
        __syncthreads();                                 // every thread is done reading h before it becomes m
        if (active && !skip) {                           // step 4: damped weights
            const double ssum = sh_ssum[kk];
            for (int i = e0; i < N; i += estride) {
                const double r = __ddiv_rn(B[i], ssum);
                double v;
                if (r <= 0.0) v = 0.0;
                else if (r >= 1.0) v = 1.0;
                else v = damp_pow(__ddiv_rn(__dsub_rn(1.0, r), -log(r)), alpha);
                A[i] = v;
            }
        }
        __syncthreads();
        if (own >= 0 && !skip) {                         // step 5
            const double total = refine_prefix(A, cum, N, lo, hi);
            if (lane == 0) sh_delta[own] = __ddiv_rn(total, static_cast<double>(N));
        }
        __syncthreads();
        if (active) {                                    // step 6: the new edges
            double* Eng = new_edges + static_cast<size_t>(k) * (N + 1);
            const double delta = skip ? 0.0 : sh_delta[kk];
            for (int j = e0; j <= N; j += estride) {
                double v;
                if (skip) v = E[j];
                else if (j == 0) v = 0.0;
                else if (j == N) v = 1.0;
                else {
                    const double t = __dmul_rn(static_cast<double>(j), delta);
                    int a = 0, b = N - 1;                // smallest i in [0, N-1] with cum[i+1] >= t, else N-1
                    while (a < b) {
                        const int mid = (a + b) >> 1;
                        if (cum[mid + 1] >= t) b = mid; else a = mid + 1;
                    }
                    v = __dadd_rn(E[a], __dmul_rn(__ddiv_rn(__dsub_rn(t, cum[a]), A[a]), __dsub_rn(E[a + 1], E[a])));
                }
                B[j] = v;
                Eng[j] = v;
            }
        }
        __syncthreads();
        if (active && !skip) {                           // step 7 check
            int bad = 0;
            for (int j = e0; j < N; j += estride)
                if (!(B[j] < B[j + 1])) bad = 1;
            if (bad) sh_bad = 1;
        }
        __syncthreads();                                 // the shared arrays are reused by the next pass
    }
    const int bad = sh_bad;
    if (threadIdx.x == 0) {
        if (bad) status[0] += 1;                         // refinements rejected since the host last collected
        status[2] = bad;                                 // outcome of the most recent refinement
    }
    const int cells = d * N;
    if (bad) {                                           // grid and table stay as they were; H too, unless this is the fused
        if (clear_hist_always)                           // step (the next step's iteration starts from clean accumulators)
            for (int c = threadIdx.x; c < cells; c += blockDim.x) hist[c] = 0.0;
        return;
    }
    const bool one_pass = d <= group;                    // every dimension's new edges are still in shared memory (B)
    const double* smd = reinterpret_cast<const double*>(smem);
    for (int c = threadIdx.x; c < cells; c += blockDim.x) {
        const int k = c / N, i = c - k * N;
        const double* En = one_pass ? smd + static_cast<size_t>(k) * per_dim + (N + 1) : new_edges + static_cast<size_t>(k) * (N + 1);
        const double lo_e = one_pass ? En[i] : __ldcg(En + i);          // written by other warps of this CTA
        const double hi_e = one_pass ? En[i + 1] : __ldcg(En + i + 1);
        write_table_cell(table, precision, static_cast<size_t>(c), lo_e, __dsub_rn(hi_e, lo_e));
        hist[c] = 0.0;
    }
    for (int e = threadIdx.x; e < d * (N + 1); e += blockDim.x) {
        const int k = e / (N + 1), j = e - k * (N + 1);
        edges[e] = one_pass ? smd[static_cast<size_t>(k) * per_dim + (N + 1) + j] : __ldcg(new_edges + e);
    }
}

__global__ void refine_kernel(double* edges, double* hist, int N, double alpha, double* new_edges, int d, void* table,
                              int precision, int* status, int smem_bytes)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    refine_all(edges, hist, N, alpha, new_edges, d, table, precision, status, smem_raw, static_cast<size_t>(smem_bytes), false);
}

// ------------------------------------------------------------------------------------------------
// debug_events_kernel: the parity hook.  One thread per event, same process_event as iterate_kernel,
// table read from global memory.
// ------------------------------------------------------------------------------------------------
template <class F, int D>
__global__ void debug_events_kernel(const __grid_constant__ IterArgs a, int32_t* __restrict__ bins,
                                    double* __restrict__ x, double* __restrict__ jac, double* __restrict__ f,
                                    double* __restrict__ wf, int32_t* __restrict__ pass)
{
    using real = typename F::real;
    const uint32_t idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= a.count) return;
    const int d = D ? D : a.dim;
    real J, fv;
    bool ps;
    const double w = process_event<F, D>(
        a, a.e_lo_first + idx, a.table,
        [&](int k, int i, real xv) {
            bins[static_cast<size_t>(idx) * d + k] = i;
            x[static_cast<size_t>(idx) * d + k] = static_cast<double>(xv);
        },
        J, fv, ps);
    jac[idx] = static_cast<double>(J);
    f[idx] = static_cast<double>(fv);
    wf[idx] = w;
    pass[idx] = ps ? 1 : 0;
}

}  // namespace vegas
