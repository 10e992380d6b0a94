// gbfit.cu -- kernels and C ABI of the GB waveform + delta-lnL hot path for sm_100a (B200).
//
// Launch structure of one call (all on the caller's stream, no host synchronisation):
//   1. cudaMemsetAsync of the work counters
//   2. gb_prep_kernel      one thread per proposal row: per-source constants (step O1) for the new and/or
//                          old source plus the row's walker / PSD row / move (one 192-byte record per side),
//                          classification by (window length N, swap?, fast or general slow part) and
//                          warp-aggregated append to that class's work list
//   3. gb_main_kernel<N,SWAP,FAST>  one persistent launch per class that can occur: a group of G threads (one
//                          CTA) takes rows of the class's list by a global ticket (taken three items ahead; the
//                          next record arrives by cp.async while the current row computes), evaluates the slow
//                          part at N time samples (O2-O5; gb_fast.cuh, or gb_math.cuh for rows outside its
//                          limits), runs the length-N FFT of A and E in shared memory (O6; gb_fft.cuh), and
//                          finishes in the same kernel with either the waveform store, the inner products +
//                          delta lnL / overlap (O7, O8) or the atomic scatter into the residual (O9).  Waveforms
//                          never touch global memory on the delta-lnL / update paths.
// gb_band_sweep and gb_temper_sweep (Algorithms 1 and 2 of the paper) have their own kernels, gb_band.cuh and
// gb_temper.cuh, built from the same slow part and FFT.
#include <cuda_runtime.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>
#include <mutex>

#include <vector>

#include "../../include/gbfit.h"
#include "gb_fast.cuh"
#include "gb_fft.cuh"
#include "gb_math.cuh"
#include "gb_tables.hpp"

using namespace gbk;

namespace {

// tunables (defaults chosen from A/B runs on B200, see profiles/README.md)
#ifndef GB_TPSM
#define GB_TPSM 512        // resident threads per SM the main kernels are register-limited to (launch bounds)
#endif
#ifndef GB_ORBIT_PREFETCH
#define GB_ORBIT_PREFETCH 1   // request the orbit rows of sample j+1 before evaluating sample j
#endif
#ifndef GB_L2_PREFETCH
#define GB_L2_PREFETCH 1      // delta lnL: request the next item's residual / PSD window into L2
#endif
#ifndef GB_SWAP_BATCH
#define GB_SWAP_BATCH 4       // SWAP / overlap epilogue: window bins per thread whose loads are in flight together
#endif
#ifndef GB_EPI_BATCH
#define GB_EPI_BATCH 8        // delta-lnL epilogue: window bins per thread whose loads are in flight together
#endif
#ifndef GB_STREAM_LOADS
#define GB_STREAM_LOADS 1     // window loads bypass L1 allocation
#endif
#ifndef GB_WARP_SYNC
#define GB_WARP_SYNC 1        // one-warp groups (N = 128, 256) use __syncwarp instead of the CTA barrier
#endif
#ifndef GB_BAND_GM
#define GB_BAND_GM 2          // band / ladder kernels: threads per task = GB_BAND_GM x the FFT group (the slow part, the
#endif                        // staging and the inner products use all of them, the FFT the first group)
#ifndef GB_UNROLL
#define GB_UNROLL 1        // unroll factor of the per-thread time-sample loop
#endif

enum Mode { MODE_WAVEFORM = 0, MODE_DLNL = 1, MODE_UPDATE = 2, MODE_OVERLAP = 3 };   // OVERLAP: SWAP kernels, no residual
constexpr int kNumClasses = 16;  // class = 4 * log2(N / 128) + 2 * general + swap  (general: outside the fast path)

// ------------------------------------------------------------------------------------------------ args
struct PrepArgs {
    const double* params_new;
    const double* params_old;
    const int32_t* walker_index;
    const int8_t* move;
    const uint8_t* accepted;
    const int32_t* n_bins;
    const int32_t* walker_psd;
    int move_all, N, mode, n_walkers, n_psd, keep;
    int Nmax;                // MODE_WAVEFORM: row pitch of AE_out (a row with N_b > Nmax is a row error)
    int64_t B;
    double Tobs, tau, Rmax;  // Rmax = AU / c
    int64_t kmax;            // largest valid global bin (Nyquist)
    SrcConst* src_new;
    SrcConst* src_old;
    int32_t* lists;          // [kNumClasses][B]
    int32_t* counts;         // [kNumClasses]
    int32_t* errflag;
    double* dlnL_out;
    // gb_delta_loglike_accept: per-row (beta, logq, logu) packed for the main kernels; the work lists are binned by
    // (class, walker chunk): accept = 1 counts the rows of every bin, accept = 2 is the full pass appending at the bins' offsets
    int accept;
    int K;                   // walker chunks
    const int32_t* chunk_first;   // DEVICE [K]: first walker of every chunk (gb_chunk_bounds_kernel)
    const double* logq;
    const double* logu;
    const double* beta;
    double4* accpar;         // [B] (beta, logq, logu, -)
    int32_t* bin_count;      // [kNumClasses * K] rows per bin (pass 1)
    const int32_t* bin_off;  // [kNumClasses * K] exclusive prefix sum of bin_count
    int32_t* bin_cursor;     // [kNumClasses * K] rows appended so far (pass 2)
    uint8_t* accepted_out;
};

// One accepted row of gb_delta_loglike_accept: where its window sits in the store and where it goes.
struct alignas(16) KeptEnt {
    int64_t off;             // element offset of the window in the store: [2][N] complex128
    int64_t kmin;            // global bin of window bin 0
    int32_t walker;
    int32_t N;               // 0: empty slot
    double sgn;              // r += sgn * h   (ADD: -1, REMOVE: +1)
};
static_assert(sizeof(KeptEnt) == 32, "KeptEnt layout");

struct MainArgs {
    const SrcConst* src_new;
    const SrcConst* src_old;
    const int32_t* lists;
    const int32_t* counts;
    int32_t* counters;       // [kNumClasses] next-item tickets
    const double* orbit;     // [11][N] for this class's N
    const cx* tw;            // [1024]
    int64_t B;
    int mode;
    // data view
    double* resid;
    const double* psd;
    const int32_t* walker_psd;
    int64_t k_lo, n_f;
    int32_t n_walkers, n_psd, psd_is_inverse;
    // proposals
    const int32_t* walker_index;
    const int8_t* move;
    int move_all;
    // outputs
    double* dlnL_out;
    double* aux_out;
    double* AE_out;
    int64_t* kmin_out;
    int Nmax;
    double Tobs, tau;
    cx* wkeep;               // gb_delta_loglike_keep: every row's window goes here (class base + list position)
    int64_t wkeep_cap;       // capacity in elements
    int32_t* errflag;
    // gb_delta_loglike_accept (ACC instantiations): the epilogue decides beta dlnL + logq >= logu and stores the ACCEPTED
    // windows into wkeep, one KeptEnt per accepted row in a global list; store slots and list positions are reserved a few
    // at a time per CTA.  The rows are binned by (class, walker chunk); a launch works on one bin.
    KeptEnt* ent;
    int64_t ent_cap;
    const double4* accpar;
    uint8_t* accepted_out;
    unsigned long long* store_cursor;   // next free element of wkeep
    int32_t* ent_cursor;                // next free list position
    int32_t* sc_claim;                  // fused update: pieces handed out to CTAs so far
    const struct Piece* pieces;         // fused update: the accepted windows of EARLIER walker chunks (complete), cut up
    const int32_t* n_pieces;            //               and how many there are (fixed during a launch)
    const int32_t* bin_count;
    const int32_t* bin_off;
    int32_t* bin_ticket;
    // DIRECT instantiations: the proposal arrays themselves (thread 0 of a CTA does step O1 of its rows)
    const double* params_new;
    const double* params_old;
    double Rmax;
    int64_t kmax;
    int K, chunk;
    int pool_r;                         // store slots / list positions a CTA reserves at a time
    int fuse;                           // != 0: CTAs move accepted windows of earlier chunks into the residual between items
};

// element offset of a class's region of the kept windows: the classes before it, count x 2 N each
__device__ __forceinline__ int64_t keep_class_base(const int32_t* counts, int cls) {
    int64_t base = 0;
    for (int c = 0; c < cls; c++) base += (int64_t)counts[c] * 2 * (128 << (c >> 2));
    return base;
}

// ------------------------------------------------------------------------------------------------ prep
__device__ __forceinline__ int class_of_N(int N) {
    return N == 128 ? 0 : N == 256 ? 1 : N == 512 ? 2 : N == 1024 ? 3 : -1;
}

__global__ void __launch_bounds__(256) gb_prep_kernel(PrepArgs a) {
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int cls = -1;
    int bin = -1;           // accept mode: cls * K + walker chunk
    bool use_old = false;   // the row's single source is the OLD one (REMOVE)
    const bool count_only = a.accept == 1;
    if (b < a.B) {
        const int mv = a.mode == MODE_WAVEFORM ? GB_ADD : (a.move ? (int)a.move[b] : a.move_all);
        const int N = a.n_bins ? a.n_bins[b] : a.N;
        const int cN = class_of_N(N);
        bool ok = cN >= 0 && mv >= GB_ADD && mv <= GB_SWAP && !((a.keep || a.accept) && mv == GB_SWAP);
        if (a.mode == MODE_WAVEFORM && N > a.Nmax) ok = false;                 // would overrun the row of AE_out
        if (mv != GB_REMOVE && !a.params_new) ok = false;                      // per-row move needs a side that is NULL
        if (mv != GB_ADD && !a.params_old) ok = false;
        int w = 0, prow = 0;
        if (a.mode == MODE_OVERLAP) {          // walker_index carries the PSD row itself (NULL: row 0)
            prow = a.walker_index ? a.walker_index[b] : 0;
            ok = ok && prow >= 0 && prow < a.n_psd;
        } else if (a.mode != MODE_WAVEFORM) {
            w = a.walker_index[b];
            ok = ok && w >= 0 && w < a.n_walkers;
            if (ok) prow = a.walker_psd ? a.walker_psd[w] : (a.n_psd == 1 ? 0 : w);
            ok = ok && prow >= 0 && prow < a.n_psd;
        }
        const bool active = a.accepted ? a.accepted[b] != 0 : true;
        if (!ok) {
            if (!count_only) {
                atomicOr(a.errflag, 1);
                if (a.dlnL_out) a.dlnL_out[b] = __longlong_as_double(0x7ff8000000000000LL);
                if (a.accept) a.accepted_out[b] = 0;
            }
        } else if (active) {
            bool fast = true;
            if (mv != GB_REMOVE) fast = fast && fast_path_ok(a.params_new + 8 * b, a.Tobs, a.tau, a.Rmax);
            if (mv != GB_ADD) fast = fast && fast_path_ok(a.params_old + 8 * b, a.Tobs, a.tau, a.Rmax);
            cls = 4 * cN + (fast ? 0 : 2) + (mv == GB_SWAP ? 1 : 0);
            use_old = mv == GB_REMOVE;
            if (a.accept) {   // walker chunk: the last k with chunk_first[k] <= w
                int k = 0;
                while (k + 1 < a.K && a.chunk_first[k + 1] <= w) k++;
                bin = cls * a.K + k;
            }
            if (!count_only) {
                if (a.accept) a.accpar[b] = make_double4(a.beta ? a.beta[b] : 1.0, a.logq ? a.logq[b] : 0.0, a.logu[b], 0.0);
                if (mv != GB_REMOVE) {
                    SrcConst s;
                    source_constants(a.params_new + 8 * b, a.Tobs, a.tau, N, s);
                    s.fast = fast_path_ok(a.params_new + 8 * b, a.Tobs, a.tau, a.Rmax) ? 1 : 0;
                    s.walker = w;  s.psd_row = prow;  s.move = mv;
                    if (s.kmin + N - 1 > a.kmax) atomicOr(a.errflag, 2);
                    a.src_new[b] = s;
                }
                if (mv != GB_ADD) {
                    SrcConst s;
                    source_constants(a.params_old + 8 * b, a.Tobs, a.tau, N, s);
                    s.fast = fast_path_ok(a.params_old + 8 * b, a.Tobs, a.tau, a.Rmax) ? 1 : 0;
                    s.walker = w;  s.psd_row = prow;  s.move = mv;
                    if (s.kmin + N - 1 > a.kmax) atomicOr(a.errflag, 2);
                    a.src_old[b] = s;
                }
            }
        }
    }
    const unsigned lane = threadIdx.x & 31;
    if (a.accept) {   // binned lists: one atomic per (warp, bin); pass 1 counts, pass 2 appends at the bin's offset
        const unsigned listed = __ballot_sync(0xffffffffu, bin >= 0);
        if (bin >= 0) {
            const unsigned m = __match_any_sync(listed, bin);
            const int leader = __ffs(m) - 1;
            int base = 0;
            if ((int)lane == leader) base = atomicAdd((count_only ? a.bin_count : a.bin_cursor) + bin, __popc(m));
            base = __shfl_sync(m, base, leader);
            if (!count_only)
                a.lists[a.bin_off[bin] + base + __popc(m & ((1u << lane) - 1))] = (int32_t)b | (use_old ? (int32_t)0x80000000 : 0);
        }
        return;
    }
    // warp-aggregated append: one atomic per (warp, class)
#pragma unroll
    for (int c = 0; c < kNumClasses; c++) {
        const unsigned m = __ballot_sync(0xffffffffu, cls == c);
        if (m == 0) continue;
        const int leader = __ffs(m) - 1;
        int base = 0;
        if ((int)lane == leader) base = atomicAdd(a.counts + c, __popc(m));
        base = __shfl_sync(0xffffffffu, base, leader);
        if (cls == c) a.lists[(int64_t)c * a.B + base + __popc(m & ((1u << lane) - 1))] = (int32_t)b | (use_old ? (int32_t)0x80000000 : 0);
    }
}

// gb_delta_loglike_accept, before the binning: rows per walker of THIS batch ...
__global__ void __launch_bounds__(256) gb_walker_hist_kernel(const int32_t* __restrict__ walker_index, int64_t B, int n_walkers,
                                                             int32_t* hist) {
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int w = b < B ? walker_index[b] : -1;
    const bool ok = w >= 0 && w < n_walkers;
    const unsigned m0 = __ballot_sync(0xffffffffu, ok);
    if (ok) {
        const unsigned m = __match_any_sync(m0, w);
        if ((int)(threadIdx.x & 31) == __ffs(m) - 1) atomicAdd(hist + w, __popc(m));
    }
}
// ... and the walker chunks cut from it: chunk sizes (in ROWS) fall off geometrically, ratio 3/4.  The accepted rows of
// chunk c are moved into the residual while chunk c + 1 is evaluated, about one 4 KB piece per evaluated row, so a chunk
// must not be much smaller than the one before it; and what the last chunk accepts is left to the closing launch, so the
// last chunk is the smallest.  A batch that touches only some of the walkers is cut by the rows it has, not by walker index.
// row_start[k] = rows of the batch in the chunks before k (the binned lists of chunk k start there, see run_call)
__global__ void gb_chunk_bounds_kernel(const int32_t* __restrict__ hist, int n_walkers, int K, int64_t B, int32_t* chunk_first,
                                       int32_t* row_start) {
    double total = 0.0, sz = 1.0;
    for (int k = 0; k < K; k++, sz *= 0.75) total += sz;
    int64_t rows = 0;
    for (int w = 0; w < n_walkers; w++) rows += hist[w];
    double cum = 0.0;
    sz = 1.0;
    int w = 0;
    int64_t seen = 0;
    for (int k = 0; k < K; k++, sz *= 0.75) {
        const int64_t target = (int64_t)(cum / total * (double)rows + 0.5);   // rows before chunk k
        while (w < n_walkers && seen < target) seen += hist[w++];
        chunk_first[k] = k == 0 ? 0 : w;
        row_start[k] = (int32_t)seen;
        cum += sz;
    }
}

// One-pass binning: the list of bin (class, chunk k) may hold every row of chunk k, so it starts at class * B + row_start[k]
// and no counting pass is needed (the lists have room for B rows per class)
__global__ void gb_bin_off_kernel(const int32_t* __restrict__ row_start, int64_t B, int K, int32_t* off) {
    const int i = threadIdx.x;
    if (i < kNumClasses * K) off[i] = (int32_t)((i / K) * B + (row_start ? row_start[i % K] : 0));
}

// exclusive prefix sum of the bin counts (one thread: at most 16 x 16 bins)
__global__ void gb_bin_scan_kernel(const int32_t* __restrict__ count, int32_t* off, int n) {
    int acc = 0;
    for (int i = 0; i < n; i++) {
        off[i] = acc;
        acc += count[i];
    }
}

// ------------------------------------------------------------------------------------------------ main
// barrier of a group of G threads (the first G threads of the CTA, whole warps): a one-warp group only needs the
// warp-level barrier; larger groups use named barrier 1 with a thread count, so that in the band / ladder kernels
// (whose CTAs are wider than the FFT group) the first G threads can run the FFT while the others wait at cta_sync
// (the SWAP kernels run two groups side by side, one per waveform: group g uses named barrier 1 + g)
template <int G>
__device__ __forceinline__ void group_sync(int bar = 1) {
#if GB_WARP_SYNC
    if (G == 32) __syncwarp();
    else asm volatile("bar.sync %0, %1;" ::"r"(bar), "n"(G) : "memory");
#else
    asm volatile("bar.sync %0, %1;" ::"r"(bar), "n"(G) : "memory");
#endif
}
// barrier of the H threads that transform ONE channel (the FFT stages of A and E never touch each other's buffer): a
// warp-level barrier when the channel is one warp or less (N <= 512), else a named barrier of its own
template <int H>
__device__ __forceinline__ void chan_sync(int id) {
    if (H <= 32) __syncwarp();
    else asm volatile("bar.sync %0, %1;" ::"r"(id), "n"(H) : "memory");
}
// barrier of the whole CTA of T threads (barrier 0)
template <int T>
__device__ __forceinline__ void cta_sync() {
    if (T == 32) __syncwarp();
    else __syncthreads();
}

// FFT of both channels of one item: threads [0, G/2) transform A, threads [G/2, G) transform E (gb_fft.cuh).
//   fft_store: every stage written back, the buffers end up holding the window in natural order;
//   fft_regs:  the last stage stays in registers, h[m] = bin ht + (G/2) m of this thread's channel.
#define GB_STAGE_X(N_, R_, Ns_)                                       \
    {                                                                 \
        StageRegs<N_, R_> rg;                                         \
        fft_stage_read<N_, R_>(buf, ht, rg);                          \
        chan_sync<Plan<N_>::G / 2>(cbar);                             \
        fft_stage_compute<N_, R_, Ns_>(tw, ht, rg);                   \
        fft_stage_store<N_, R_, Ns_>(buf, ht, rg);                    \
        chan_sync<Plan<N_>::G / 2>(cbar);                             \
    }
#define GB_STAGE_L(N_, R_, Ns_)                                       \
    {                                                                 \
        StageRegs<N_, R_> rg;                                         \
        fft_stage_read<N_, R_>(buf, ht, rg);                          \
        fft_stage_compute<N_, R_, Ns_>(tw, ht, rg);                   \
        fft_last_to_bins<N_, R_>(rg, h);                              \
    }
template <int N>
__device__ __forceinline__ void fft_store(cx* bA, cx* bE, const cx* __restrict__ tw, int tid, int bar = 1) {
    constexpr int H = Plan<N>::G / 2;
    cx* buf = tid < H ? bA : bE;
    const int ht = tid < H ? tid : tid - H;
    const int cbar = 3 + 2 * (bar - 1) + (tid < H ? 0 : 1);   // named barrier of this group's channel (ids 3 .. 6)
    if constexpr (N == 128) { GB_FFT_PLAN_128(GB_STAGE_X, GB_STAGE_X) }
    if constexpr (N == 256) { GB_FFT_PLAN_256(GB_STAGE_X, GB_STAGE_X) }
    if constexpr (N == 512) { GB_FFT_PLAN_512(GB_STAGE_X, GB_STAGE_X) }
    if constexpr (N == 1024) { GB_FFT_PLAN_1024(GB_STAGE_X, GB_STAGE_X) }
}
template <int N>
__device__ __forceinline__ void fft_regs(cx* bA, cx* bE, const cx* __restrict__ tw, int tid, cx* h) {
    constexpr int H = Plan<N>::G / 2;
    cx* buf = tid < H ? bA : bE;
    const int ht = tid < H ? tid : tid - H;
    const int cbar = 3 + (tid < H ? 0 : 1);
    if constexpr (N == 128) { GB_FFT_PLAN_128(GB_STAGE_X, GB_STAGE_L) }
    if constexpr (N == 256) { GB_FFT_PLAN_256(GB_STAGE_X, GB_STAGE_L) }
    if constexpr (N == 512) { GB_FFT_PLAN_512(GB_STAGE_X, GB_STAGE_L) }
    if constexpr (N == 1024) { GB_FFT_PLAN_1024(GB_STAGE_X, GB_STAGE_L) }
}

// orbit table rows at sample n (coalesced across the group; the table stays L1/L2 resident)
template <int N, bool FAST>
struct OrbitRegs;
template <int N>
struct OrbitRegs<N, true> {
    OrbitSampleAB o;
    __device__ __forceinline__ void load(const double* __restrict__ orbit, int n) {
        o.Rx = __ldg(orbit + 0 * N + n);
        o.Ry = __ldg(orbit + 1 * N + n);
#pragma unroll
        for (int d = 0; d < 3; d++) {
            o.a[d] = __ldg(orbit + (2 + d) * N + n);
            o.b[d] = __ldg(orbit + (5 + d) * N + n);
        }
    }
    __device__ __forceinline__ void eval(const SrcConst& s, double t, double nfrac, double tau, double scale, cd& As,
                                         cd& Es) const {
        slow_sample_fast(s, o, t, nfrac, tau, scale, As, Es);
    }
};
template <int N>
struct OrbitRegs<N, false> {
    OrbitSample o;
    __device__ __forceinline__ void load(const double* __restrict__ orbit, int n) {
        o.Rx = __ldg(orbit + 0 * N + n);
        o.Ry = __ldg(orbit + 1 * N + n);
#pragma unroll
        for (int d = 0; d < 3; d++) {
            o.a[d] = __ldg(orbit + (2 + d) * N + n);
            o.b[d] = __ldg(orbit + (5 + d) * N + n);
            o.c[d] = __ldg(orbit + (8 + d) * N + n);
        }
    }
    __device__ __forceinline__ void eval(const SrcConst& s, double t, double nfrac, double tau, double scale, cd& As,
                                         cd& Es) const {
        slow_sample(s, o, t, nfrac, tau, scale, As, Es);
    }
};

// slow part at this thread's samples n = tid + G j: bA, bE receive (-1)^n T/(2N) (A_s, E_s)(t_n); after
// fft_all they hold the window, element j <-> global bin kmin + j.  s_src is the group's shared copy of the
// source record (already visible to the whole group).  The orbit rows of sample j+1 are requested before
// sample j is evaluated.
template <int N, int G, bool FAST>
__device__ __forceinline__ void slow_part(const SrcConst* s_src, const double* __restrict__ orbit, cx* bA, cx* bE,
                                          double Tobs, double tau, int tid, int bar = 1) {
    constexpr int S = N / G;
    const double dtN = Tobs / (double)N;
    const double scale = (tid & 1) ? -Tobs / (2.0 * N) : Tobs / (2.0 * N);   // G is even: parity of n = parity of tid
    OrbitRegs<N, FAST> nxt;
    nxt.load(orbit, tid);
    constexpr int kUnroll = GB_UNROLL;
#pragma unroll kUnroll
    for (int j = 0; j < S; j++) {
        const int n = tid + G * j;
#if GB_ORBIT_PREFETCH
        const OrbitRegs<N, FAST> cur = nxt;
        if (j + 1 < S) nxt.load(orbit, n + G);
#else
        if (j > 0) nxt.load(orbit, n);
        const OrbitRegs<N, FAST>& cur = nxt;
#endif
        cd As, Es;
        cur.eval(*s_src, (double)n * dtN, (double)n * (1.0 / N), tau, scale, As, Es);
        bA[pad_idx<N>(n)] = {As.re, As.im};
        bE[pad_idx<N>(n)] = {Es.re, Es.im};
    }
    group_sync<G>(bar);
}

// sum NV per-thread values over the group; result valid in thread 0
template <int G, int NV>
__device__ __forceinline__ void group_reduce(double* v, double* s_red, int tid) {
#pragma unroll
    for (int i = 0; i < NV; i++) {
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) v[i] += __shfl_xor_sync(0xffffffffu, v[i], off);
    }
    if (G > 32) {
        const int warp = tid >> 5;
        if ((tid & 31) == 0) {
#pragma unroll
            for (int i = 0; i < NV; i++) s_red[warp * NV + i] = v[i];
        }
        group_sync<G>();
        if (tid == 0) {
#pragma unroll
            for (int w = 1; w < G / 32; w++) {
#pragma unroll
                for (int i = 0; i < NV; i++) v[i] += s_red[w * NV + i];
            }
        }
        group_sync<G>();
    }
}

// One batch of window bins of ONE channel: residual r and weight 1/S_n at elements i_first + H c (the
// non-SWAP epilogue, fed from registers).  Same load policy as WinBatch below.
template <int CH>
struct WinBatch1 {
    cx r[CH];
    double w[CH];
    template <int H, bool CHECK>
    __device__ __forceinline__ void load(const double* __restrict__ rC, const double* __restrict__ SC, int64_t i_first,
                                         int64_t n_f, bool inv) {
        bool ok[CH];
#pragma unroll
        for (int c = 0; c < CH; c++) {
            const int64_t i = i_first + H * c;
            ok[c] = CHECK ? (i >= 0 && i < n_f) : true;   // !CHECK: the whole window lies inside the stored band
            const int64_t ic = ok[c] ? i : 0;
#if GB_STREAM_LOADS
            const double2 a2 = __ldcg(reinterpret_cast<const double2*>(rC + 2 * ic));
            w[c] = __ldcg(SC + ic);
#else
            const double2 a2 = *reinterpret_cast<const double2*>(rC + 2 * ic);
            w[c] = SC[ic];
#endif
            r[c] = {a2.x, a2.y};
        }
        if (!inv) {
#pragma unroll
            for (int c = 0; c < CH; c++) w[c] = 1.0 / w[c];
        }
#pragma unroll
        for (int c = 0; c < CH; c++) {
            if (!ok[c]) {
                w[c] = 0.0;
                r[c] = {0.0, 0.0};
            }
        }
    }
};

// One batch of window bins of a thread: residual (A, E) and weights 1/S_n (A, E) at elements i_first + G c.
// The loads are unconditional (index clamped, values zeroed when the bin lies outside the stored band) so
// that all of them are in flight together, and they are cached in L2 only (ld.global.cg): the orbit tables
// and twiddles, re-read by every item, keep the L1.
template <int CH>
struct WinBatch {
    cx ra[CH], re[CH];
    double wa[CH], we[CH];
    template <int G, bool CHECK>
    __device__ __forceinline__ void load(const double* __restrict__ rA, const double* __restrict__ rE,
                                         const double* __restrict__ SA, const double* __restrict__ SE, int64_t i_first,
                                         int64_t n_f, bool inv) {
        bool ok[CH];
#pragma unroll
        for (int c = 0; c < CH; c++) {
            const int64_t i = i_first + G * c;
            ok[c] = CHECK ? (i >= 0 && i < n_f) : true;   // !CHECK: the whole window lies inside the stored band
            const int64_t ic = ok[c] ? i : 0;
#if GB_STREAM_LOADS
            const double2 a2 = __ldcg(reinterpret_cast<const double2*>(rA + 2 * ic));
            const double2 e2 = __ldcg(reinterpret_cast<const double2*>(rE + 2 * ic));
            wa[c] = __ldcg(SA + ic);
            we[c] = __ldcg(SE + ic);
#else
            const double2 a2 = *reinterpret_cast<const double2*>(rA + 2 * ic);
            const double2 e2 = *reinterpret_cast<const double2*>(rE + 2 * ic);
            wa[c] = SA[ic];
            we[c] = SE[ic];
#endif
            ra[c] = {a2.x, a2.y};
            re[c] = {e2.x, e2.y};
        }
        if (!inv) {
#pragma unroll
            for (int c = 0; c < CH; c++) {
                wa[c] = 1.0 / wa[c];
                we[c] = 1.0 / we[c];
            }
        }
#pragma unroll
        for (int c = 0; c < CH; c++) {
            if (!ok[c]) {
                wa[c] = we[c] = 0.0;
                ra[c] = re[c] = {0.0, 0.0};
            }
        }
    }
    // weights only (gb_overlap has no residual): r = 0
    template <int G>
    __device__ __forceinline__ void load_weights(const double* __restrict__ SA, const double* __restrict__ SE,
                                                 int64_t i_first, int64_t n_f, bool inv) {
#pragma unroll
        for (int c = 0; c < CH; c++) {
            const int64_t i = i_first + G * c;
            const bool ok = i >= 0 && i < n_f;
            const int64_t ic = ok ? i : 0;
            const double sa = __ldcg(SA + ic), se = __ldcg(SE + ic);
            wa[c] = ok ? (inv ? sa : 1.0 / sa) : 0.0;
            we[c] = ok ? (inv ? se : 1.0 / se) : 0.0;
            ra[c] = re[c] = {0.0, 0.0};
        }
    }
};
// FP64 add into the residual, resolved in L2, no return value.  Spelled out in PTX: atomicAdd(double*) on a pointer whose
// address space the compiler cannot prove compiles to a generic ATOM with a compare-and-swap fallback loop
// (gb_temper_kernel<128> did), and with a fence behind it to ATOMG instead of RED.
__device__ __forceinline__ void red_add_f64(double* p, double v) {
    asm volatile("red.global.add.f64 [%0], %1;" ::"l"(__cvta_generic_to_global(p)), "d"(v) : "memory");
}
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int K>
__device__ __forceinline__ void cp_async_wait() {
    asm volatile("cp.async.wait_group %0;" ::"n"(K) : "memory");
}

constexpr int kRecChunks = (int)(sizeof(SrcConst) / 16);   // 16-byte pieces of one source record

// ---- fused update of gb_delta_loglike_accept -------------------------------------------------------------------
__device__ __forceinline__ int ld_acquire_s32(const int32_t* p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ int ld_relaxed_s32(const int32_t* p) {
    int v;
    asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// entries and windows were written by other CTAs of the same launch: read them through L2 (an L1 line may predate them)
__device__ __forceinline__ KeptEnt load_ent(const KeptEnt* p) {
    const longlong2 a = __ldcg(reinterpret_cast<const longlong2*>(p));
    const int4 b = __ldcg(reinterpret_cast<const int4*>(p) + 1);
    KeptEnt e;
    e.off = a.x;
    e.kmin = a.y;
    e.walker = b.x;
    e.N = b.y;
    e.sgn = __hiloint2double(b.w, b.z);
    return e;
}

// r[walker] += sgn * window for one accepted row (step O9), by T threads: the window is read from the store
// (coalesced 16-byte loads, four in flight per thread) and added with FP64 atomics resolved in L2.
template <int T>
__device__ __forceinline__ void scatter_entry(const KeptEnt& e, const cx* __restrict__ store, double* resid, int64_t k_lo,
                                              int64_t n_f, int tid) {
    const int N = e.N;
    const cx* w = store + e.off;
    double* r = resid + (size_t)e.walker * 2 * (size_t)n_f * 2;
    const int64_t i0 = e.kmin - k_lo;
    const double sgn = e.sgn;
    const bool inband = i0 >= 0 && i0 + N <= n_f;
    for (int x0 = tid; x0 < 2 * N; x0 += 4 * T) {
        double2 h[4];
#pragma unroll
        for (int u = 0; u < 4; u++) {
            const int x = x0 + u * T;
            h[u] = x < 2 * N ? __ldcg(reinterpret_cast<const double2*>(w + x)) : make_double2(0.0, 0.0);
        }
#pragma unroll
        for (int u = 0; u < 4; u++) {
            const int x = x0 + u * T;
            if (x < 2 * N) {
                const int ch = x >= N ? 1 : 0;
                const int64_t i = i0 + (x - ch * N);
                if (inband || (i >= 0 && i < n_f)) {
                    double* p = r + ((size_t)ch * (size_t)n_f + (size_t)i) * 2;
                    atomicAdd(p, sgn * h[u].x);
                    atomicAdd(p + 1, sgn * h[u].y);
                }
            }
        }
    }
}

// ---- bulk asynchronous copies (TMA without a tensor map) for the fused update ------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_test(unsigned long long* bar, unsigned parity) {
    unsigned ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
// (the stored windows are read exactly once: L2 evict-first, so that they do not push out the residual lines the
// evaluation shares between neighbouring rows)
__device__ __forceinline__ void bulk_load(void* smem_dst, const void* gsrc, unsigned bytes, unsigned long long* bar) {
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
                     smem_u32(smem_dst)),
                 "l"(gsrc), "r"(bytes), "r"(smem_u32(bar)), "l"(pol)
                 : "memory");
}
__device__ __forceinline__ void bulk_reduce_add_f64(void* gdst, const void* smem_src, unsigned bytes) {
    asm volatile("cp.reduce.async.bulk.global.shared::cta.bulk_group.add.f64 [%0], [%1], %2;" ::"l"(gdst), "r"(smem_u32(smem_src)),
                 "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }

// Fused update of gb_delta_loglike_accept, one small state machine per CTA, driven by thread 0 at two checkpoints of
// every item.  The call works through the walkers in K chunks; while the rows of chunk c+1 are evaluated, the accepted
// windows of chunks <= c -- complete, and read by no row any more -- move from the store into the residual.  Between two
// chunks gb_pieces_kernel cuts the new windows into PIECES of at most kPieceElems elements (one 4 KB staging buffer per
// CTA) with their clipped destinations worked out, so that the code inside the evaluation loop is a few dozen
// instructions: a piece goes into the staging buffer with one bulk copy (completion on an mbarrier) and from there into
// the walker's residual row with one bulk REDUCTION per channel (cp.reduce.async.bulk ... add.f64: the adds happen in L2,
// no thread waits for them, no register of the evaluation is involved).  Pieces are claimed four at a time.
constexpr int kPieceElems = 256;   // complex elements of a piece = of the staging buffer
constexpr int kScQueue = 4;
struct alignas(16) Piece {
    unsigned long long src;    // element offset of the piece in the store
    unsigned long long dst;    // element offset in the residual array of the first segment's first bin
    unsigned nload;            // bytes to copy store -> staging buffer
    unsigned nb;               // bytes of a segment (after clipping to the stored band)
    unsigned s0;               // byte offset of segment 0 in the staging buffer
    unsigned s1;               // byte offset of segment 1 (the E channel of a window that fits in one piece), 0: none
};
static_assert(sizeof(Piece) == 32, "Piece layout");
struct ScState {
    unsigned long long mbar;
    Piece q[kScQueue];     // claimed pieces
    Piece cur;             // the piece in flight
    int q_n, q_pos;        // pieces in q; the next one to start
    int state;             // 0: buffer free, 1: bulk load in flight, 2: bulk reductions in flight
    unsigned parity;       // phase of mbar the load in flight completes
    int n_pieces;          // pieces that exist for this launch (fixed)
    int exhausted;         // nothing left to claim
    // this CTA's reservations for the rows it accepts
    long long pool_off;    // next free store slot (a window of this launch's N)
    int pool_left;
    int ent_next, ent_left;   // next free list position
};
__device__ __forceinline__ void sc_init(ScState& s, int n_pieces) {
    mbar_init(&s.mbar, 1);
    s.q_n = s.q_pos = s.state = 0;
    s.parity = 0;
    s.n_pieces = n_pieces;
    s.exhausted = n_pieces <= 0;
    s.pool_off = 0;
    s.pool_left = s.ent_next = s.ent_left = 0;
}
// first checkpoint of an item (after the slow part): a piece that has landed goes on into the residual
__device__ __forceinline__ void sc_reduce_if_landed(const MainArgs& a, ScState& s, cx* stage) {
    if (s.state != 1 || !mbar_test(&s.mbar, s.parity)) return;
    s.parity ^= 1u;
    double* dst = a.resid + 2 * s.cur.dst;
    char* src = reinterpret_cast<char*>(stage);
    if (s.cur.nb) {
        bulk_reduce_add_f64(dst, src + s.cur.s0, s.cur.nb);
        if (s.cur.s1) bulk_reduce_add_f64(dst + 2 * a.n_f, src + s.cur.s1, s.cur.nb);   // the E row follows the A row
    }
    bulk_commit();
    s.state = 2;
}
// second checkpoint (end of the item): free the buffer, start the next piece
__device__ __forceinline__ void sc_next_piece(const MainArgs& a, ScState& s, cx* stage) {
    if (s.state == 1) return;            // still loading
    if (s.state == 2) {
        bulk_wait_read0();               // the staging buffer has been read (the adds complete on their own)
        s.state = 0;
    }
    if (s.q_pos >= s.q_n) {
        if (s.exhausted) return;
        // a plain fetch-and-add: positions at or beyond n_pieces are taken by nobody (gb_pieces_kernel pulls the counter back)
        const int i = atomicAdd(a.sc_claim, kScQueue);
        if (i >= s.n_pieces) {
            s.exhausted = 1;
            return;
        }
        const int n = min(kScQueue, s.n_pieces - i);
        for (int k = 0; k < n; k++) {
            const uint4* p = reinterpret_cast<const uint4*>(a.pieces + i + k);
            const uint4 lo = __ldcg(p), hi = __ldcg(p + 1);
            reinterpret_cast<uint4*>(&s.q[k])[0] = lo;
            reinterpret_cast<uint4*>(&s.q[k])[1] = hi;
        }
        s.q_n = n;
        s.q_pos = 0;
        fence_proxy_async();   // the windows were written with ordinary stores (by earlier launches); bulk copies read them
    }
    s.cur = s.q[s.q_pos++];
    mbar_expect_tx(&s.mbar, s.cur.nload);
    bulk_load(stage, a.wkeep + s.cur.src, s.cur.nload, &s.mbar);
    s.state = 1;
}
// Between two walker chunks of gb_delta_loglike_accept: the accepted rows listed since the last time (positions
// [*ent_done, *ent_cursor), all written by finished launches) are cut into pieces for the fused update.
struct PiecesArgs {
    const KeptEnt* ent;
    Piece* pieces;
    int64_t pieces_cap, ent_cap;
    const int32_t* ent_cursor;
    const int32_t* ent_done;
    int32_t* piece_cursor;
    int64_t k_lo, n_f;
    int32_t n_walkers;
};

__global__ void __launch_bounds__(256) gb_pieces_kernel(PiecesArgs a) {
    int64_t hi = *a.ent_cursor;
    if (hi > a.ent_cap) hi = a.ent_cap;
    for (int64_t i = *a.ent_done + (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < hi; i += (int64_t)gridDim.x * blockDim.x) {
        const KeptEnt e = a.ent[i];
        if (e.N <= 0 || e.walker < 0 || e.walker >= a.n_walkers) continue;
        const int N = e.N;
        const int64_t i0 = e.kmin - a.k_lo;
        if (2 * N <= kPieceElems) {   // the whole window (A then E) is one piece
            const int64_t jlo = max((int64_t)0, -i0), jhi = min((int64_t)N, a.n_f - i0);
            if (jhi <= jlo) continue;
            const int pos = atomicAdd(a.piece_cursor, 1);
            if (pos >= a.pieces_cap) continue;
            Piece p;
            p.src = (unsigned long long)e.off;
            p.dst = (unsigned long long)((int64_t)e.walker * 2 * a.n_f + i0 + jlo);
            p.nload = 2u * N * 16u;
            p.nb = (unsigned)(jhi - jlo) * 16u;
            p.s0 = (unsigned)jlo * 16u;
            p.s1 = (unsigned)(N + jlo) * 16u;
            a.pieces[pos] = p;
        } else {                      // pieces of kPieceElems bins of one channel
            const int per = N / kPieceElems;
            for (int q = 0; q < 2 * per; q++) {
                const int ch = q / per;
                const int64_t x0 = (int64_t)(q % per) * kPieceElems;
                const int64_t jlo = max(x0, -i0), jhi = min(x0 + kPieceElems, a.n_f - i0);
                if (jhi <= jlo) continue;
                const int pos = atomicAdd(a.piece_cursor, 1);
                if (pos >= a.pieces_cap) continue;
                Piece p;
                p.src = (unsigned long long)(e.off + (int64_t)ch * N + x0);
                p.dst = (unsigned long long)(((int64_t)e.walker * 2 + ch) * a.n_f + i0 + jlo);
                p.nload = kPieceElems * 16u;
                p.nb = (unsigned)(jhi - jlo) * 16u;
                p.s0 = (unsigned)(jlo - x0) * 16u;
                p.s1 = 0;
                a.pieces[pos] = p;
            }
        }
    }
}

// ... and then published: CTAs that found nothing to claim ran the claim counter past the end; it is pulled back first
__global__ void gb_ready_kernel(const int32_t* ent_cursor, int32_t* ent_done, const int32_t* piece_cursor, int32_t* sc_claim,
                                int32_t* n_pieces) {
    if (*sc_claim > *n_pieces) *sc_claim = *n_pieces;
    *n_pieces = *piece_cursor;
    *ent_done = *ent_cursor;
}

// Work distribution: items of a class are handed out by a global ticket counter, in list order, so the CTAs
// that run at the same time work on neighbouring rows -- consecutive sources of one walker -- and share that
// walker's residual in L2 (a fixed round-robin deal lets the CTAs drift apart and more than doubles the DRAM
// traffic).  The ticket is taken three items ahead, its list entry is read two items ahead, the 192-byte
// source record(s) of the next item are copied into the other half of s_src with cp.async while the current
// item computes, and (delta lnL) the next item's residual / PSD window is requested into L2 one whole item
// before its inner products read it: no global-memory round trip is exposed between items.
// A list entry is the row index, with bit 31 set when the row's single source is the OLD one (REMOVE);
// -1 marks the end of the list.
// VAR: 0 = the batched kernels; 1 = gb_delta_loglike_accept; 2 = DIRECT, the one-launch path of small uniform batches (no
// prep kernel, no work lists: CTA c takes rows c, c + gridDim.x, ... and thread 0 works out each row's record itself)
// SWAP kernels: a CTA is TWO groups of G threads that compute the two waveforms of a row side by side (group 0 the old
// source, group 1 the new one, each with its own buffers and named barrier) and share the inner products: the same
// shared-memory footprint per CTA as one group doing them one after the other, but twice the threads, so the SM holds 16
// warps instead of 12 and a row takes half as long.
template <int N, bool SWAP, bool FAST, int VAR>
__global__ void __launch_bounds__(Plan<N>::G*(SWAP ? 2 : 1), GB_TPSM / (Plan<N>::G * (SWAP ? 2 : 1))) gb_main_kernel(MainArgs a) {
    constexpr int G = Plan<N>::G;
    constexpr int T = SWAP ? 2 * G : G;   // threads of the CTA
    constexpr int S = N / G;
    constexpr int PN = padded_len<N>();
    constexpr int NS = SWAP ? 2 : 1;
    constexpr int cls = 4 * (N == 128 ? 0 : N == 256 ? 1 : N == 512 ? 2 : 3) + (FAST ? 0 : 2) + (SWAP ? 1 : 0);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cx* bufA0 = reinterpret_cast<cx*>(smem_raw);      // first (or only) waveform
    cx* bufE0 = bufA0 + PN;
    cx* bufA1 = bufE0 + PN;                           // SWAP: the new source; first = old
    cx* bufE1 = bufA1 + PN;
    __shared__ __align__(16) SrcConst s_src[2][NS];   // [buffer][0 = old or only, 1 = new (SWAP)]
    __shared__ double s_red[(T / 32) * 5 + 1];

    __shared__ int s_ent[2];
    __shared__ int s_pos[2];   // list positions of the entries in s_ent (gb_delta_loglike_keep)
    __shared__ __align__(16) double4 s_par[2];   // (beta, logq, logu) of the item in each buffer (gb_delta_loglike_accept)
    __shared__ long long s_off;                  // store offset of this item's window, -1: rejected

    const int tid = threadIdx.x;
    const int grp = SWAP ? tid / G : 0;      // SWAP: which waveform this thread computes
    const int lt = SWAP ? tid - grp * G : tid;
    auto item_sync = [&]() {                 // barrier of all threads that work on the item
        if (SWAP) __syncthreads();
        else group_sync<G>();
    };
    constexpr bool accept = VAR == 1 && !SWAP;   // gb_delta_loglike_accept (its own instantiation: the plain kernels carry none of it)
    constexpr bool direct = VAR == 2 && !SWAP;   // one-launch path of small batches
    const int bin = accept ? cls * a.K + a.chunk : cls;   // accept: the lists are binned by (class, walker chunk)
    const int count = direct ? (int)((a.B - blockIdx.x + gridDim.x - 1) / gridDim.x)   // rows of THIS CTA
                             : accept ? a.bin_count[bin] : a.counts[cls];
    int32_t* const ticket = accept ? a.bin_ticket + bin : a.counters + cls;
    int direct_next = 0;   // (thread 0, direct) this CTA's next private ticket
    auto take = [&](int n) {
        if (direct) {
            const int t = direct_next;
            direct_next += n;
            return t;
        }
        return atomicAdd(ticket, n);
    };
    // fused update (thread 0 only): accepted windows of earlier walker chunks travel store -> staging buffer -> residual as
    // bulk asynchronous copies / reductions; no other thread and no register of the evaluation is involved
    cx* stage = reinterpret_cast<cx*>(smem_raw) + 2 * PN;
    __shared__ ScState s_scs;
    const bool fuse = accept && a.fuse;
    if (accept && tid == 0) sc_init(s_scs, fuse ? *a.n_pieces : 0);
    auto finish = [&]() {   // before the CTA exits: what it claimed is finished, list positions it did not use are marked empty
        if (accept && tid == 0) {
            if (fuse) {
                s_scs.exhausted = 1;
                for (;;) {
                    if (s_scs.state == 1) {
                        while (!mbar_test(&s_scs.mbar, s_scs.parity)) {}
                        sc_reduce_if_landed(a, s_scs, stage);
                    }
                    if (s_scs.state == 0 && s_scs.q_pos >= s_scs.q_n) break;
                    sc_next_piece(a, s_scs, stage);
                }
                asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
            }
            KeptEnt none;
            none.off = 0;  none.kmin = 0;  none.walker = 0;  none.N = 0;  none.sgn = 0.0;
            for (int i = 0; i < s_scs.ent_left; i++)
                if (s_scs.ent_next + i < a.ent_cap) a.ent[s_scs.ent_next + i] = none;
        }
    };
    if (!accept && count == 0) return;   // (accept: one exit at the end, so that the closing code exists once)
    const int32_t* __restrict__ list = accept ? a.lists + a.bin_off[bin] : a.lists + (int64_t)cls * a.B;
    // ticket -> list entry (row index, bit 31: the row's single source is the OLD one), -1 past the end
    auto entry_of = [&](int t) -> int {
        if (t >= count) return -1;
        if (direct) return (int)(blockIdx.x + (int64_t)t * gridDim.x) | (a.move_all == GB_REMOVE ? (int)0x80000000 : 0);
        return __ldg(list + t);
    };

    auto fetch = [&](int entry, int bufi) {
        const int64_t row = entry & 0x7fffffff;
        if (direct) {   // step O1 and the row checks of gb_prep_kernel, by thread 0 (move < 0 marks a row error)
            if (tid == 0) {
                const double* p = (entry < 0 ? a.params_old : a.params_new) + 8 * row;
                SrcConst s;
                source_constants(p, a.Tobs, a.tau, N, s);
                s.fast = fast_path_ok(p, a.Tobs, a.tau, a.Rmax) ? 1 : 0;
                s.move = a.move_all;
                int w = 0, prow = 0;
                bool ok = true;
                if (a.mode != MODE_WAVEFORM) {
                    w = a.walker_index[row];
                    ok = w >= 0 && w < a.n_walkers;
                    if (ok) prow = a.walker_psd ? a.walker_psd[w] : (a.n_psd == 1 ? 0 : w);
                    ok = ok && prow >= 0 && prow < a.n_psd;
                }
                s.walker = w;
                s.psd_row = prow;
                if (!ok) s.move = -1;
                else if (s.kmin + N - 1 > a.kmax) atomicOr(a.errflag, 2);
                s_src[bufi][0] = s;
            }
            return;
        }
        if (SWAP) {
            if (tid < kRecChunks)
                cp_async16(reinterpret_cast<char*>(&s_src[bufi][0]) + 16 * tid,
                           reinterpret_cast<const char*>(a.src_old + row) + 16 * tid);
            else if (tid < 2 * kRecChunks)
                cp_async16(reinterpret_cast<char*>(&s_src[bufi][NS - 1]) + 16 * (tid - kRecChunks),
                           reinterpret_cast<const char*>(a.src_new + row) + 16 * (tid - kRecChunks));
        } else if (tid < kRecChunks) {
            const SrcConst* g = (entry < 0 ? a.src_old : a.src_new) + row;
            cp_async16(reinterpret_cast<char*>(&s_src[bufi][0]) + 16 * tid, reinterpret_cast<const char*>(g) + 16 * tid);
        } else if (accept && tid < kRecChunks + 2) {
            cp_async16(reinterpret_cast<char*>(&s_par[bufi]) + 16 * (tid - kRecChunks),
                       reinterpret_cast<const char*>(a.accpar + row) + 16 * (tid - kRecChunks));
        }
    };

    int t_nx2 = 0;   // (thread 0) ticket of the item after next
    if (tid == 0) {
        const int t = take(3);
        s_ent[0] = entry_of(t);
        s_ent[1] = entry_of(t + 1);
        s_pos[0] = t;
        s_pos[1] = t + 1;
        t_nx2 = t + 2;
    }
    item_sync();
    int e_cur = s_ent[0], e_nxt = s_ent[1];
    int pos_cur = s_pos[0], pos_nxt = s_pos[1];
    const int64_t keep_base = (a.wkeep && !accept) ? keep_class_base(a.counts, cls) : 0;
    if (!accept && e_cur == -1) return;
    int buf = 0;
    if (e_cur != -1) {
        fetch(e_cur, 0);
        cp_async_commit();
    }

    while (e_cur != -1) {
        const bool has_nxt = e_nxt != -1;
        if (has_nxt) fetch(e_nxt, buf ^ 1);
        cp_async_commit();
        cp_async_wait<1>();            // this item's record(s) have landed (the next item's may be in flight)
        item_sync();
        const SrcConst* rec = s_src[buf];
        const int64_t b = e_cur & 0x7fffffff;
        const int mv = rec[0].move;
        const bool bad_row = direct && mv < 0;   // (direct) walker / PSD row out of range: NaN, nothing computed
        if (bad_row && tid == 0) {
            atomicOr(a.errflag, 1);
            if (a.dlnL_out) a.dlnL_out[b] = __longlong_as_double(0x7ff8000000000000LL);
        }

        // ---- waveform(s)
        if (direct) {
            if (!bad_row) {
                if (rec[0].fast) slow_part<N, G, true>(&rec[0], a.orbit, bufA0, bufE0, a.Tobs, a.tau, tid);
                else slow_part<N, G, false>(&rec[0], a.orbit, bufA0, bufE0, a.Tobs, a.tau, tid);
            }
        } else if (SWAP) {   // group 0: the old source into buffers 0, group 1: the new one into buffers 1
            slow_part<N, G, FAST>(&rec[grp ? NS - 1 : 0], a.orbit, grp ? bufA1 : bufA0, grp ? bufE1 : bufE0, a.Tobs, a.tau, lt, 1 + grp);
        } else {
            slow_part<N, G, FAST>(&rec[0], a.orbit, bufA0, bufE0, a.Tobs, a.tau, tid);
        }
        // (thread 0) next ticket and the list entry of the ticket taken one item ago: issued here, after the
        // register-hungry slow part, and consumed at the end of the item, behind the FFT and the epilogue
        int t_nx3 = 0, e_nx2 = -1;
        if (tid == 0) {
            t_nx3 = take(1);
            e_nx2 = entry_of(t_nx2);
        }
        // fused update, first checkpoint of the item: move the piece in flight one stage on
        if (fuse && tid == 0) sc_reduce_if_landed(a, s_scs, stage);
        const int64_t kmin0 = rec[0].kmin;

        // ---- ask L2 for the next item's residual / PSD window
        if (GB_L2_PREFETCH && a.mode == MODE_DLNL && has_nxt) {
            cp_async_wait<0>();
            item_sync();
            const SrcConst& nx = s_src[buf ^ 1][NS - 1];
            const int64_t i0 = nx.kmin - a.k_lo;
            const size_t nf = (size_t)a.n_f;
            const bool nx_bad = direct && nx.move < 0;   // (direct) a row error: its walker / PSD row are not valid indices
            const size_t nxw = nx_bad ? 0 : (size_t)nx.walker, nxp = nx_bad ? 0 : (size_t)nx.psd_row;
            const double* rAn = a.resid + (nxw * 2 + 0) * nf * 2;
            const double* rEn = a.resid + (nxw * 2 + 1) * nf * 2;
            const double* SAn = a.psd + (nxp * 2 + 0) * nf;
            const double* SEn = a.psd + (nxp * 2 + 1) * nf;
            if (i0 >= 0 && i0 + N + 16 <= a.n_f) {           // window (plus the line it may end in) is stored
                const double* pA = rAn + 2 * (i0 + 8 * tid);
                const double* pE = rEn + 2 * (i0 + 8 * tid);
#pragma unroll
                for (int l = 0; l <= N / 8; l += T) {      // 128-byte lines of the complex128 windows
                    if (l + tid <= N / 8) {
                        prefetch_l2(pA + 16 * l);
                        prefetch_l2(pE + 16 * l);
                    }
                }
                const double* pSA = SAn + i0 + 16 * tid;
                const double* pSE = SEn + i0 + 16 * tid;
#pragma unroll
                for (int l = 0; l <= N / 16; l += T) {     // and of the f64 PSD windows
                    if (l + tid <= N / 16) {
                        prefetch_l2(pSA + 16 * l);
                        prefetch_l2(pSE + 16 * l);
                    }
                }
            } else {
                for (int l = tid; l <= N / 8; l += T) {
                    const int64_t i = i0 + 8 * l;
                    if (i >= 0 && i < a.n_f) {
                        prefetch_l2(rAn + 2 * i);
                        prefetch_l2(rEn + 2 * i);
                    }
                }
                for (int l = tid; l <= N / 16; l += T) {
                    const int64_t i = i0 + 16 * l;
                    if (i >= 0 && i < a.n_f) {
                        prefetch_l2(SAn + i);
                        prefetch_l2(SEn + i);
                    }
                }
            }
        }

        // ---- FFT: SWAP keeps both windows in shared memory; otherwise the last stage stays in registers,
        //      h[m] = bin ht + H m of this thread's channel (threads [0, H): A, [H, G): E)
        constexpr int H = G / 2, M = N / H;
        cx h[M];
        if (SWAP) {
            fft_store<N>(grp ? bufA1 : bufA0, grp ? bufE1 : bufE0, a.tw, lt, 1 + grp);
            __syncthreads();   // both windows are complete
        } else {
            fft_regs<N>(bufA0, bufE0, a.tw, tid, h);
        }
        const int ch = tid >= H ? 1 : 0;
        const int ht = tid - ch * H;

        // ---- epilogue
        if (bad_row) {
        } else if (a.mode == MODE_WAVEFORM) {
            double2* outA = reinterpret_cast<double2*>(a.AE_out) + ((size_t)b * 2 + 0) * (size_t)a.Nmax;
            double2* outE = reinterpret_cast<double2*>(a.AE_out) + ((size_t)b * 2 + 1) * (size_t)a.Nmax;
#pragma unroll
            for (int m = 0; m < M; m++) (ch ? outE : outA)[ht + H * m] = make_double2(h[m].re, h[m].im);
            if (tid == 0 && a.kmin_out) a.kmin_out[b] = kmin0;
        } else {
            const int w = rec[0].walker;
            const size_t nf = (size_t)a.n_f;
            double* rA = a.resid + ((size_t)w * 2 + 0) * nf * 2;
            double* rE = a.resid + ((size_t)w * 2 + 1) * nf * 2;
            const int64_t i0w = kmin0 - a.k_lo;                         // residual element of window bin 0
            const bool inband0 = i0w >= 0 && i0w + N <= a.n_f;          // the whole window is stored
            if (a.mode == MODE_DLNL || a.mode == MODE_OVERLAP) {
                const int prow = rec[0].psd_row;
                const double* SA = a.psd + ((size_t)prow * 2 + 0) * nf;
                const double* SE = a.psd + ((size_t)prow * 2 + 1) * nf;
                const bool inv = a.psd_is_inverse != 0;
                const double norm = 4.0 / a.Tobs;
                constexpr int ST = N / T;                        // SWAP: bins per thread (both channels), all T threads
                constexpr int CH = SWAP ? (ST < GB_SWAP_BATCH ? ST : GB_SWAP_BATCH) : (S < 4 ? S : 4);   // bins per thread whose loads are in flight together
                if (!SWAP) {
                    // this thread's channel: bins ht + H m (consecutive threads, consecutive bins)
                    const double* rC = ch ? rE : rA;
                    const double* SC = ch ? SE : SA;
                    constexpr int CH1 = GB_EPI_BATCH < M ? GB_EPI_BATCH : M;      // bins per thread whose loads are in flight together
                    double v[2] = {0.0, 0.0};   // <h|h>, <r|h>
#pragma unroll
                    for (int m0 = 0; m0 < M; m0 += CH1) {
                        WinBatch1<CH1> wb;
                        if (inband0) wb.template load<H, false>(rC, SC, i0w + ht + H * m0, a.n_f, inv);
                        else wb.template load<H, true>(rC, SC, i0w + ht + H * m0, a.n_f, inv);
#pragma unroll
                        for (int c = 0; c < CH1; c++) {
                            const cx hc = h[m0 + c], rc = wb.r[c];
                            v[0] += wb.w[c] * (hc.re * hc.re + hc.im * hc.im);
                            v[1] += wb.w[c] * (rc.re * hc.re + rc.im * hc.im);
                        }
                    }
                    if (a.wkeep && !accept) {   // keep the window for gb_residual_update_kept: [position][channel][N]
                        const int64_t off = keep_base + (int64_t)pos_cur * 2 * N + (int64_t)ch * N + ht;
                        if (off - ht - (int64_t)ch * N + 2 * N <= a.wkeep_cap) {
#pragma unroll
                            for (int m = 0; m < M; m++) a.wkeep[off + H * m] = h[m];
                        } else if (tid == 0) {
                            atomicOr(a.errflag, 4);
                        }
                    }
                    group_reduce<G, 2>(v, s_red, tid);
                    if (tid == 0) {
                        const double hh = norm * v[0], rh = norm * v[1];
                        const double dl = (mv == GB_REMOVE ? -rh : rh) - 0.5 * hh;
                        a.dlnL_out[b] = dl;
                        if (a.aux_out) {
                            a.aux_out[2 * b] = hh;
                            a.aux_out[2 * b + 1] = rh;
                        }
                        if (accept) {   // Eq. 13 in log form, each operation rounded on its own (as the oracle)
                            const double4 par = s_par[buf];
                            bool acc = __dadd_rn(__dmul_rn(par.x, dl), par.y) >= par.z;
                            long long off = -1;
                            if (acc) {
                                ScState& sc = s_scs;
                                if (sc.pool_left == 0) {   // reserve store slots and list positions for the next few accepted rows
                                    const int R = a.pool_r;
                                    sc.pool_off = (long long)atomicAdd(a.store_cursor, (unsigned long long)(R * 2 * N));
                                    sc.ent_next = atomicAdd(a.ent_cursor, R);
                                    sc.pool_left = sc.ent_left = R;
                                }
                                if (sc.pool_off + 2 * N > a.wkeep_cap || sc.ent_next >= a.ent_cap) {   // store full: the row cannot be applied
                                    atomicOr(a.errflag, 4);
                                    acc = false;
                                } else {
                                    off = sc.pool_off;
                                    KeptEnt e;
                                    e.off = off;
                                    e.kmin = kmin0;
                                    e.walker = w;
                                    e.N = N;
                                    e.sgn = 1.0;   // the sign of the move is in the stored window
                                    a.ent[sc.ent_next] = e;
                                    sc.pool_off += 2 * N;
                                    sc.pool_left--;
                                    sc.ent_next++;
                                    sc.ent_left--;
                                }
                            }
                            a.accepted_out[b] = acc ? 1 : 0;
                            s_off = off;
                        }
                    }
                    if (accept) {
                        group_sync<G>();
                        const long long off = s_off;
                        if (off >= 0) {
                            cx* dst = a.wkeep + off + (int64_t)ch * N + ht;
                            const double sg = mv == GB_REMOVE ? 1.0 : -1.0;   // the store holds the CHANGE of the residual
#pragma unroll
                            for (int m = 0; m < M; m++)   // streaming stores: read back once, much later -- not worth L2 lines
                                __stcs(reinterpret_cast<double2*>(dst + H * m), make_double2(sg * h[m].re, sg * h[m].im));
                        }
                    }
                } else {
                    // buffers: 0 = old (o), 1 = new (a)
                    const int64_t kmin1 = rec[NS - 1].kmin;
                    const int64_t shift = kmin1 - kmin0;   // o index of a's bin j is j + shift
                    const int64_t i1w = kmin1 - a.k_lo;
                    const bool inband1 = i1w >= 0 && i1w + N <= a.n_f;
                    double v[5] = {0.0, 0.0, 0.0, 0.0, 0.0};   // aa, ra, ao, oo, ro
#pragma unroll
                    for (int m0 = 0; m0 < ST; m0 += CH) {
                        WinBatch<CH> wn, wo;   // the new source's window and the old one's (equal when shift == 0)
                        if (a.mode == MODE_OVERLAP) {      // no residual: weights only
                            wn.template load_weights<T>(SA, SE, i1w + tid + T * m0, a.n_f, inv);
                            wo.template load_weights<T>(SA, SE, i0w + tid + T * m0, a.n_f, inv);
                        } else if (inband0 && inband1) {
                            wn.template load<T, false>(rA, rE, SA, SE, i1w + tid + T * m0, a.n_f, inv);
                            if (shift != 0) wo.template load<T, false>(rA, rE, SA, SE, i0w + tid + T * m0, a.n_f, inv);
                            else wo = wn;
                        } else {
                            wn.template load<T, true>(rA, rE, SA, SE, i1w + tid + T * m0, a.n_f, inv);
                            wo.template load<T, true>(rA, rE, SA, SE, i0w + tid + T * m0, a.n_f, inv);
                        }
#pragma unroll
                        for (int c = 0; c < CH; c++) {
                            const int j = tid + T * (m0 + c);
                            const cx oa = bufA0[pad_idx<N>(j)], oe = bufE0[pad_idx<N>(j)];   // the old window at bin j
                            {
                                const cx ha = bufA1[pad_idx<N>(j)], he = bufE1[pad_idx<N>(j)];
                                const cx ra = wn.ra[c], re = wn.re[c];
                                const double wa = wn.wa[c], we = wn.we[c];
                                v[0] += wa * (ha.re * ha.re + ha.im * ha.im) + we * (he.re * he.re + he.im * he.im);
                                v[1] += wa * (ra.re * ha.re + ra.im * ha.im) + we * (re.re * he.re + re.im * he.im);
                                cx sa = oa, se = oe;   // ... and at the bin under a's bin j (the same one when the windows coincide)
                                bool in = true;
                                if (shift != 0) {      // uniform over the CTA
                                    const int64_t jo = j + shift;
                                    in = jo >= 0 && jo < N;
                                    if (in) {
                                        sa = bufA0[pad_idx<N>((int)jo)];
                                        se = bufE0[pad_idx<N>((int)jo)];
                                    }
                                }
                                if (in) v[2] += wa * (ha.re * sa.re + ha.im * sa.im) + we * (he.re * se.re + he.im * se.im);
                            }
                            {
                                const cx ra = wo.ra[c], re = wo.re[c];
                                const double wa = wo.wa[c], we = wo.we[c];
                                v[3] += wa * (oa.re * oa.re + oa.im * oa.im) + we * (oe.re * oe.re + oe.im * oe.im);
                                v[4] += wa * (ra.re * oa.re + ra.im * oa.im) + we * (re.re * oe.re + re.im * oe.im);
                            }
                        }
                    }
                    group_reduce<T, 5>(v, s_red, tid);
                    if (tid == 0) {
                        const double aa = norm * v[0], ra = norm * v[1], ao = norm * v[2], oo = norm * v[3],
                                     ro = norm * v[4];
                        if (a.mode == MODE_OVERLAP) {   // <a|c> / sqrt(<a|a><c|c>), 0 when a norm vanishes
                            a.dlnL_out[b] = (aa > 0.0 && oo > 0.0) ? ao / sqrt(aa * oo) : 0.0;
                            if (a.aux_out) {
                                a.aux_out[2 * b] = aa;
                                a.aux_out[2 * b + 1] = oo;
                            }
                        } else {
                            a.dlnL_out[b] = -0.5 * (aa + oo - 2.0 * ao - 2.0 * ra + 2.0 * ro);
                            if (a.aux_out) {
                                a.aux_out[2 * b] = aa;
                                a.aux_out[2 * b + 1] = ra;
                            }
                        }
                    }
                }
            } else {   // MODE_UPDATE: r -= a (ADD), r += h (REMOVE), r += o - a (SWAP)
                const double sgn0 = SWAP ? 1.0 : (mv == GB_REMOVE ? 1.0 : -1.0);
                if (!SWAP) {
                    double* rC = (ch ? rE : rA) + 2 * (i0w + ht);
                    if (inband0) {            // common case: no per-bin range checks
#pragma unroll
                        for (int m = 0; m < M; m++) {
                            atomicAdd(rC + 2 * H * m, sgn0 * h[m].re);
                            atomicAdd(rC + 2 * H * m + 1, sgn0 * h[m].im);
                        }
                    } else {
#pragma unroll
                        for (int m = 0; m < M; m++) {
                            const int64_t i = i0w + ht + H * m;
                            if (i >= 0 && i < a.n_f) {
                                atomicAdd(rC + 2 * H * m, sgn0 * h[m].re);
                                atomicAdd(rC + 2 * H * m + 1, sgn0 * h[m].im);
                            }
                        }
                    }
                } else
#pragma unroll
                for (int m = 0; m < N / T; m++) {
                    const int j = tid + T * m;
                    int64_t i = kmin0 + j - a.k_lo;
                    if (i >= 0 && i < a.n_f) {
                        const cx ha = bufA0[pad_idx<N>(j)], he = bufE0[pad_idx<N>(j)];
                        atomicAdd(rA + 2 * i, sgn0 * ha.re);
                        atomicAdd(rA + 2 * i + 1, sgn0 * ha.im);
                        atomicAdd(rE + 2 * i, sgn0 * he.re);
                        atomicAdd(rE + 2 * i + 1, sgn0 * he.im);
                    }
                    if (SWAP) {
                        i = rec[NS - 1].kmin + j - a.k_lo;
                        if (i >= 0 && i < a.n_f) {
                            const cx ha = bufA1[pad_idx<N>(j)], he = bufE1[pad_idx<N>(j)];
                            atomicAdd(rA + 2 * i, -ha.re);
                            atomicAdd(rA + 2 * i + 1, -ha.im);
                            atomicAdd(rE + 2 * i, -he.re);
                            atomicAdd(rE + 2 * i + 1, -he.im);
                        }
                    }
                }
            }
        }
        if (tid == 0) {
            s_ent[0] = e_nx2;
            s_pos[0] = t_nx2;
            t_nx2 = t_nx3;
        }
        item_sync();   // the waveform buffers, s_red and this half of s_src are reused from here on
        if (fuse && tid == 0) sc_next_piece(a, s_scs, stage);   // second checkpoint of the item
        if (!has_nxt) break;
        e_cur = e_nxt;
        e_nxt = s_ent[0];
        pos_cur = pos_nxt;
        pos_nxt = s_pos[0];
        buf ^= 1;
    }
    finish();
}

// One waveform of the band / ladder kernels: slow part by all G threads of the CTA, FFT (every stage written back) by the
// first PG.  Deliberately NOT inlined: those kernels generate waveforms at several places (cache fill, old and new source,
// fast and general slow part) and their hot loops are bound by instruction fetch (17 % of the warp samples wait for
// instructions, ncu); one copy of this code, at one address, serves every call site of a kernel.
template <int N, int G, int PG>
__device__ __noinline__ void seq_window(const SrcConst* rec, const double* __restrict__ orbit, const cx* __restrict__ tw,
                                        cx* bA, cx* bE, double Tobs, double tau, int tid) {
    if (rec->fast) slow_part<N, G, true>(rec, orbit, bA, bE, Tobs, tau, tid);
    else slow_part<N, G, false>(rec, orbit, bA, bE, Tobs, tau, tid);
    if (tid < PG) fft_store<N>(bA, bE, tw, tid);
}

// Step O1 of one source by the calling thread (band / ladder kernels), out of line for the same reason
template <int N>
__device__ __noinline__ void seq_o1(const double* theta, double Tobs, double tau, double Rmax, int64_t kmax, int32_t* errflag,
                                    SrcConst* dst) {
    SrcConst s;
    source_constants(theta, Tobs, tau, N, s);
    s.fast = fast_path_ok(theta, Tobs, tau, Rmax) ? 1 : 0;
    if (s.kmin + N - 1 > kmax) atomicOr(errflag, 2);
    *dst = s;
}

#include "gb_band.cuh"
#include "gb_temper.cuh"

template <int N, bool SWAP, bool ACC = false>
constexpr size_t main_smem_bytes() {
    return (size_t)padded_len<N>() * sizeof(cx) * 2 * (SWAP ? 2 : 1) + (ACC ? (size_t)kPieceElems * sizeof(cx) : 0);
}

}  // namespace

// ------------------------------------------------------------------------------------------------ kept windows
// gb_residual_update_kept: scatter of the accepted rows from the windows gb_delta_loglike_keep left in scratch.  The
// class lists, their counts and the source records of that call are still in the context; one CTA per list entry.
struct KeptArgs {
    const int32_t* counts;
    const int32_t* lists;
    const SrcConst* src_new;
    const SrcConst* src_old;
    const cx* wkeep;
    const uint8_t* accepted;
    double* resid;
    int64_t B, k_lo, n_f;
    int64_t wkeep_cap;   // elements the keep call was allowed to write: windows past it were never stored
    int32_t n_walkers;   // of the gb_data passed to THIS call (the records carry the keep call's walker indices)
    int32_t* errflag;
    double sign;     // +1 applies the moves, -1 undoes them
};

__global__ void __launch_bounds__(128) gb_scatter_kept_kernel(KeptArgs a) {
    int64_t base = 0;
    for (int cls = 0; cls < kNumClasses; cls++) {
        const int N = 128 << (cls >> 2);
        const int count = a.counts[cls];
        const int32_t* __restrict__ list = a.lists + (int64_t)cls * a.B;
        for (int pos = blockIdx.x; pos < count; pos += gridDim.x) {
            const int e = __ldg(list + pos);
            const int64_t b = e & 0x7fffffff;
            if (a.accepted && !a.accepted[b]) continue;
            const SrcConst* rec = (e < 0 ? a.src_old : a.src_new) + b;
            const int64_t i0 = rec->kmin - a.k_lo;
            const double sgn = a.sign * (rec->move == GB_REMOVE ? 1.0 : -1.0);   // ADD: r -= a, REMOVE: r += h
            const int64_t off = base + (int64_t)pos * 2 * N;
            if (off + 2 * N > a.wkeep_cap || rec->walker < 0 || rec->walker >= a.n_walkers) {
                if (threadIdx.x == 0) atomicOr(a.errflag, off + 2 * N > a.wkeep_cap ? 4 : 1);   // never stored / foreign view
                continue;
            }
            const cx* w = a.wkeep + off;
            double* r = a.resid + (size_t)rec->walker * 2 * (size_t)a.n_f * 2;
            for (int x = threadIdx.x; x < 2 * N; x += blockDim.x) {
                const int ch = x >= N ? 1 : 0;
                const int64_t i = i0 + (x - ch * N);
                if (i >= 0 && i < a.n_f) {
                    const cx h = w[x];
                    double* p = r + ((size_t)ch * (size_t)a.n_f + (size_t)i) * 2;
                    atomicAdd(p, sgn * h.re);
                    atomicAdd(p + 1, sgn * h.im);
                }
            }
        }
        base += (int64_t)count * 2 * N;
    }
}

// ------------------------------------------------------------------------------------------------ accepted windows
// Scatter of the list positions [*lo, *hi) of the accepted-row list of gb_delta_loglike_accept from its store: what the
// fused update of the call left over (the last walker chunk), the whole list for apply = 2, and gb_residual_update_kept
// after apply = 0.  One CTA per list position at a time; unused positions (N = 0) are skipped.
struct EntArgs {
    const KeptEnt* ent;
    const cx* store;
    const int32_t* lo;        // DEVICE: first position (NULL: 0)
    const int32_t* hi;        // DEVICE: end of the list
    int64_t ent_cap;
    double* resid;
    int64_t k_lo, n_f;
    int32_t n_walkers;        // of the gb_data passed to THIS call
    int32_t* errflag;
    double sign;              // +1 applies the moves, -1 undoes them
};

__global__ void __launch_bounds__(128) gb_scatter_ent_kernel(EntArgs a) {
    const int64_t lo = a.lo ? *a.lo : 0;
    int64_t hi = *a.hi;
    if (hi > a.ent_cap) hi = a.ent_cap;
    for (int64_t i = lo + blockIdx.x; i < hi; i += gridDim.x) {
        KeptEnt e = a.ent[i];
        if (e.N <= 0) continue;
        if (e.walker < 0 || e.walker >= a.n_walkers) {   // a data view with fewer walkers than the accept call's
            if (threadIdx.x == 0) atomicOr(a.errflag, 1);
            continue;
        }
        e.sgn *= a.sign;
        scatter_entry<128>(e, a.store, a.resid, a.k_lo, a.n_f, threadIdx.x);
    }
}

// the pieces the fused update did not get to (positions [min(claim, n), n) of the piece list), by plain loads and atomics
struct RestArgs {
    const Piece* pieces;
    const cx* store;
    const int32_t* sc_claim;
    const int32_t* n_pieces;
    double* resid;
    int64_t n_f;
};
__global__ void __launch_bounds__(128) gb_scatter_pieces_kernel(RestArgs a) {
    const int n = *a.n_pieces;
    const int lo = min(*a.sc_claim, n);
    for (int i = lo + blockIdx.x; i < n; i += gridDim.x) {
        const Piece p = a.pieces[i];
        const int nel = (int)(p.nb / 16u);
        for (int x = threadIdx.x; x < nel * (p.s1 ? 2 : 1); x += blockDim.x) {
            const int seg = x >= nel ? 1 : 0, j = x - seg * nel;
            const double2 h = __ldcg(reinterpret_cast<const double2*>(a.store + p.src) + (seg ? p.s1 : p.s0) / 16u + j);
            double* d = a.resid + 2 * (p.dst + (seg ? (unsigned long long)a.n_f : 0ull) + (unsigned long long)j);
            atomicAdd(d, h.x);
            atomicAdd(d + 1, h.y);
        }
    }
}

// ------------------------------------------------------------------------------------------------ FP64 peak
// 8 independent DFMA chains per thread, registers only (gb_measure_fp64_peak)
__global__ void __launch_bounds__(128) gb_dfma_peak_kernel(double* sink, int iters, double a, double b) {
    double x[8];
#pragma unroll
    for (int i = 0; i < 8; i++) x[i] = threadIdx.x * 1e-3 + i;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int r = 0; r < 8; r++) {
#pragma unroll
            for (int i = 0; i < 8; i++) x[i] = fma(x[i], a, b);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; i++) s += x[i];
    if (s == 12345.678) sink[0] = s;   // never true: keeps the chains alive
}

// ------------------------------------------------------------------------------------------------ context
constexpr int kHostChunks = 8;
constexpr int kHostChunksAccept = 4;   // gb_delta_loglike_accept_host: fewer, larger chunks (each is a chunked call of its own)

struct gb_ctx {
    gb_config cfg;
    int num_sms;
    double* d_orbit[4];
    cx* d_tw;
    int32_t* d_counts;      // [kNumClasses] counts, [kNumClasses] counters, [1] errflag
    SrcConst* d_src_new;
    SrcConst* d_src_old;
    int32_t* d_lists;
    cx* d_band_cache;       // current-source windows of gb_band_sweep's CTAs (gb_band.cuh)
    cx* d_temper_cache;     // set sums of gb_temper_sweep's CTAs (gb_temper.cuh)
    cx* d_wkeep;            // windows kept by gb_delta_loglike_keep for gb_residual_update_kept
    int64_t cap_new, cap_old, cap_lists, cap_band_cache, cap_temper_cache, cap_wkeep;
    int64_t kept_B;         // > 0: lists, records and windows of the last gb_delta_loglike_keep call are still valid
    int64_t kept_cap;       // elements of d_wkeep that call was allowed to write (2 x its sum_n_bins)
    int kept_mode;          // 1: every window (gb_delta_loglike_keep), 2: accepted windows + entries (gb_delta_loglike_accept)
    // gb_delta_loglike_accept: counters [store cursor (2 ints), list cursor, claim, ready_end, pad (3), then per bin:
    // count, offset, append cursor, ticket], the list of accepted rows, (beta, logq, logu) per row
    int32_t* d_wk;
    KeptEnt* d_ent;
    double4* d_accpar;
    Piece* d_pieces;        // fused update: accepted windows cut into staging-buffer sized pieces
    int32_t* d_whist;       // rows per walker of the batch (walker chunks)
    int64_t cap_wk, cap_ent, cap_accpar, cap_pieces, cap_whist;
    int grid_blocks[kNumClasses];   // resident CTAs per SM * SMs, per class
    int grid_blocks_acc[kNumClasses];   // the same for the gb_delta_loglike_accept instantiations
    int grid_blocks_dir[kNumClasses];   // and for the DIRECT (one-launch) instantiations
    // staging for the *_host entry points
    void* d_stage;
    size_t cap_stage;
    // copy streams and events of the *_host forms (chunked: the copies of chunk i+1 overlap the kernels of chunk i)
    cudaStream_t s_side[3];        // the class kernels of one call are independent: they are spread over the caller's stream
    cudaEvent_t ev_fork, ev_join[3];   // and these three, so that the tail of one overlaps the start of the next
    cudaStream_t s_in, s_out;
    cudaEvent_t ev_start, ev_in[kHostChunks], ev_done[kHostChunks];
    int64_t launches;
    cx* d_static;           // device address of g_static_scratch on cfg.device (gb_band_sweep_static)
    char err[512];
};

namespace {

int set_err(gb_ctx* ctx, int code, const char* fmt, ...) {
    if (ctx) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(ctx->err, sizeof(ctx->err), fmt, ap);
        va_end(ap);
    }
    return code;
}

#define GB_CUDA(ctx, call)                                                                              \
    do {                                                                                                \
        cudaError_t e_ = (call);                                                                        \
        if (e_ != cudaSuccess)                                                                          \
            return set_err(ctx, GB_ERR_CUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_),    \
                           __FILE__, __LINE__);                                                         \
    } while (0)

template <typename T>
int ensure_cap(gb_ctx* ctx, T** ptr, int64_t* cap, int64_t need, bool exact = false) {
    if (need <= *cap) return GB_OK;
    if (*ptr) {
        GB_CUDA(ctx, cudaDeviceSynchronize());
        GB_CUDA(ctx, cudaFree(*ptr));
        *ptr = nullptr;
        *cap = 0;
    }
    const int64_t want = exact ? need : need + need / 8;   // (exact: the multi-GB window stores, sized by the caller)
    if (cudaMalloc(reinterpret_cast<void**>(ptr), (size_t)want * sizeof(T)) != cudaSuccess) {
        cudaGetLastError();
        return set_err(ctx, GB_ERR_NOMEM, "scratch allocation of %lld bytes failed", (long long)(want * sizeof(T)));
    }
    *cap = want;
    return GB_OK;
}

template <int N, bool SWAP, bool FAST, int VAR = 0>
int setup_kernel(gb_ctx* ctx) {
    constexpr int cls = 4 * (N == 128 ? 0 : N == 256 ? 1 : N == 512 ? 2 : 3) + (FAST ? 0 : 2) + (SWAP ? 1 : 0);
    const size_t smem = main_smem_bytes<N, SWAP, VAR == 1>();
    GB_CUDA(ctx, cudaFuncSetAttribute(gb_main_kernel<N, SWAP, FAST, VAR>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int nb = 0;
    GB_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, gb_main_kernel<N, SWAP, FAST, VAR>, Plan<N>::G * (SWAP ? 2 : 1), smem));
    if (nb < 1) return set_err(ctx, GB_ERR_CUDA, "kernel class %d does not fit on an SM", cls);
    (VAR == 1 ? ctx->grid_blocks_acc : VAR == 2 ? ctx->grid_blocks_dir : ctx->grid_blocks)[cls] = nb * ctx->num_sms;
    return GB_OK;
}

template <int N, bool SWAP, bool FAST, int VAR = 0>
int launch_main(gb_ctx* ctx, MainArgs& a, int64_t B, cudaStream_t st) {
    constexpr int cls = 4 * (N == 128 ? 0 : N == 256 ? 1 : N == 512 ? 2 : 3) + (FAST ? 0 : 2) + (SWAP ? 1 : 0);
    a.orbit = ctx->d_orbit[cls >> 2];
    int64_t grid = (VAR == 1 ? ctx->grid_blocks_acc : VAR == 2 ? ctx->grid_blocks_dir : ctx->grid_blocks)[cls];
    if (grid > B) grid = B;
    gb_main_kernel<N, SWAP, FAST, VAR><<<(unsigned)grid, Plan<N>::G * (SWAP ? 2 : 1), main_smem_bytes<N, SWAP, VAR == 1>(), st>>>(a);
    ctx->launches++;
    GB_CUDA(ctx, cudaGetLastError());
    return GB_OK;
}

// The class kernels of one call work on disjoint rows, so they may run concurrently: they are dealt round-robin to the
// caller's stream and three context-owned streams (fork / join with events; capturable in a CUDA graph).  Every grid is
// persistent and fills the GPU, so in effect the CTAs of the next class start as those of the current one run out of rows:
// the launch tails overlap, and launches that find an empty list cost nothing on the critical path.
struct Fan {
    gb_ctx* ctx;
    cudaStream_t main;
    bool on;
    int n;
    cudaStream_t next() {
        if (!on) return main;
        const int i = n++ & 3;
        return i == 0 ? main : ctx->s_side[i - 1];
    }
    int begin() {
        n = 0;
        if (!on) return GB_OK;
        GB_CUDA(ctx, cudaEventRecord(ctx->ev_fork, main));
        for (int i = 0; i < 3; i++) GB_CUDA(ctx, cudaStreamWaitEvent(ctx->s_side[i], ctx->ev_fork, 0));
        return GB_OK;
    }
    int end() {
        if (!on) return GB_OK;
        for (int i = 0; i < 3; i++) {
            GB_CUDA(ctx, cudaEventRecord(ctx->ev_join[i], ctx->s_side[i]));
            GB_CUDA(ctx, cudaStreamWaitEvent(main, ctx->ev_join[i], 0));
        }
        return GB_OK;
    }
};

// the fast-path kernel of a class, then the general one for the rows outside its limits (usually none:
// that launch finds an empty list and returns at once)
template <int N, bool SWAP>
int launch_pair(gb_ctx* ctx, MainArgs& a, int64_t B, Fan& fan) {
    int rc = launch_main<N, SWAP, true>(ctx, a, B, fan.next());
    if (rc) return rc;
    return launch_main<N, SWAP, false>(ctx, a, B, fan.next());
}

struct Call {
    int mode;
    const gb_data* data;
    const double* params_new;
    const double* params_old;
    const int32_t* walker_index;
    const int8_t* move;
    int move_all;
    const uint8_t* accepted;
    int N;
    const int32_t* n_bins;
    int64_t B;
    double* dlnL_out;
    double* aux_out;
    double* AE_out;
    int64_t* kmin_out;
    int Nmax;
    int keep;               // gb_delta_loglike_keep
    int64_t sum_bins;       // sum of the rows' window lengths (keep); accept: capacity of the store in window bins
    int accept;             // gb_delta_loglike_accept: 1 = decide and keep, 2 = + fused update, 3 = + update by a separate launch
    const double* logq;
    const double* logu;
    const double* beta;
    uint8_t* accepted_out;
};

constexpr int kMaxChunks = 16;           // walker chunks of gb_delta_loglike_accept
constexpr int64_t kDirectMaxRows = 8192; // batches up to this size with one window length and one move type: one launch
constexpr int kWkHeader = 8 + kMaxChunks; // ints before the per-bin arrays of d_wk (counters, then the chunks' first walkers)
constexpr int kWkInts = kWkHeader + 4 * kNumClasses * kMaxChunks;

// scatter of list positions [from the claim counter (rest) or 0 (all), list cursor) of the last gb_delta_loglike_accept call
int scatter_entries(gb_ctx* ctx, const gb_data* data, double sign, bool rest_only, cudaStream_t st) {
    EntArgs e{};
    e.ent = ctx->d_ent;
    e.store = ctx->d_wkeep;
    e.lo = rest_only ? ctx->d_wk + 5 : nullptr;   // rows listed after the last cut into pieces
    e.hi = ctx->d_wk + 2;
    e.ent_cap = ctx->cap_ent;
    e.resid = data->resid;
    e.k_lo = data->k_lo;
    e.n_f = data->n_f;
    e.n_walkers = data->n_walkers;
    e.errflag = ctx->d_counts + 2 * kNumClasses;
    e.sign = sign;
    gb_scatter_ent_kernel<<<ctx->num_sms * 16, 128, 0, st>>>(e);
    ctx->launches++;
    GB_CUDA(ctx, cudaGetLastError());
    return GB_OK;
}

int run_call(gb_ctx* ctx, const Call& c, void* stream) {
    if (!ctx) return GB_ERR_INVALID;
    if (c.B < 0 || c.B > 0x7fffffff) return set_err(ctx, GB_ERR_INVALID, "B out of range");
    if (c.B == 0) return GB_OK;
    const bool need_new = c.mode == MODE_WAVEFORM || c.move != nullptr || c.move_all != GB_REMOVE;
    const bool need_old = c.mode != MODE_WAVEFORM && (c.move != nullptr || c.move_all != GB_ADD);
    if (c.mode == MODE_OVERLAP) {
        if (!c.data || !c.data->psd || c.data->n_f <= 0 || c.data->n_psd <= 0) return set_err(ctx, GB_ERR_INVALID, "NULL / empty PSD view");
        if (!c.params_new || !c.params_old || !c.dlnL_out) return set_err(ctx, GB_ERR_INVALID, "NULL params / output");
    } else if (c.mode != MODE_WAVEFORM) {
        if (!c.data || !c.data->resid || !c.walker_index) return set_err(ctx, GB_ERR_INVALID, "NULL data / walker_index");
        if (c.mode == MODE_DLNL && (!c.data->psd || !c.dlnL_out)) return set_err(ctx, GB_ERR_INVALID, "NULL psd / dlnL_out");
        if (c.data->n_f <= 0 || c.data->n_walkers <= 0) return set_err(ctx, GB_ERR_INVALID, "empty data view");
        if (!c.move && (c.move_all < GB_ADD || c.move_all > GB_SWAP)) return set_err(ctx, GB_ERR_INVALID, "bad move_all");
        if (c.move == nullptr) {
            if (need_new && !c.params_new) return set_err(ctx, GB_ERR_INVALID, "params_new is NULL");
            if (need_old && !c.params_old) return set_err(ctx, GB_ERR_INVALID, "params_old is NULL");
        } else if (!c.params_new && !c.params_old) {
            return set_err(ctx, GB_ERR_INVALID, "params_new and params_old are NULL");
        }
    } else {
        if (!c.params_new || !c.AE_out) return set_err(ctx, GB_ERR_INVALID, "NULL params / AE_out");
    }
    if (!c.n_bins && !(c.N == 128 || c.N == 256 || c.N == 512 || c.N == 1024))
        return set_err(ctx, GB_ERR_INVALID, "N must be 128, 256, 512 or 1024");
    if (c.mode == MODE_WAVEFORM && c.Nmax < (c.n_bins ? 128 : c.N)) return set_err(ctx, GB_ERR_INVALID, "Nmax too small");

    GB_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    int rc;
    // Small uniform batches (one window length, one move type, no SWAP): ONE launch.  No prep kernel, no work lists, no
    // scratch: CTA c takes rows c, c + gridDim.x, ... and its thread 0 does step O1 and the row checks (a batch of 64
    // rows is 0.2 us of arithmetic: the call is the latency of its launches, PAPER.md:454-456 for context).
    if (c.B <= kDirectMaxRows && !c.n_bins && !c.move && !c.keep && !c.accept && !c.accepted && c.mode != MODE_OVERLAP &&
        (c.mode == MODE_WAVEFORM || c.move_all != GB_SWAP)) {
        MainArgs a{};
        a.B = c.B;
        a.mode = c.mode;
        a.tw = ctx->d_tw;
        if (c.data) {
            a.resid = c.data->resid;
            a.psd = c.data->psd;
            a.walker_psd = c.data->walker_psd;
            a.k_lo = c.data->k_lo;
            a.n_f = c.data->n_f;
            a.n_walkers = c.data->n_walkers;
            a.n_psd = c.data->n_psd;
            a.psd_is_inverse = c.data->psd_is_inverse;
        }
        a.walker_index = c.walker_index;
        a.move_all = c.mode == MODE_WAVEFORM ? GB_ADD : c.move_all;
        a.dlnL_out = c.dlnL_out;
        a.aux_out = c.aux_out;
        a.AE_out = c.AE_out;
        a.kmin_out = c.kmin_out;
        a.Nmax = c.Nmax;
        a.Tobs = ctx->cfg.Tobs;
        a.tau = ctx->cfg.armlength / kCLight;
        a.errflag = ctx->d_counts + 2 * kNumClasses;
        a.params_new = c.params_new;
        a.params_old = c.params_old;
        a.Rmax = ctx->cfg.au / kCLight;
        a.kmax = (int64_t)floor(ctx->cfg.Tobs / (2.0 * ctx->cfg.dt));
        ctx->kept_B = 0;
        switch (c.N) {
            case 128: return launch_main<128, false, true, 2>(ctx, a, c.B, st);
            case 256: return launch_main<256, false, true, 2>(ctx, a, c.B, st);
            case 512: return launch_main<512, false, true, 2>(ctx, a, c.B, st);
            default: return launch_main<1024, false, true, 2>(ctx, a, c.B, st);
        }
    }
    if (need_new && (rc = ensure_cap(ctx, &ctx->d_src_new, &ctx->cap_new, c.B))) return rc;
    if (need_old && (rc = ensure_cap(ctx, &ctx->d_src_old, &ctx->cap_old, c.B))) return rc;
    if ((rc = ensure_cap(ctx, &ctx->d_lists, &ctx->cap_lists, c.B * kNumClasses))) return rc;
    ctx->kept_B = 0;   // whatever an earlier keep call left is overwritten from here on
    if (c.keep) {
        if (c.sum_bins < 128 * c.B || c.sum_bins > 1024 * c.B) return set_err(ctx, GB_ERR_INVALID, "sum_n_bins out of range");
        if ((rc = ensure_cap(ctx, &ctx->d_wkeep, &ctx->cap_wkeep, 2 * c.sum_bins))) return rc;
    }
    // gb_delta_loglike_accept: walker chunks (the fused update of chunk c runs under the evaluation of chunk c + 1)
    const int nw = c.data ? c.data->n_walkers : 0;
    int K = 1;
    int pool_r[4] = {1, 1, 1, 1};
    int64_t store_slack = 0, ent_slack = 0;
    if (c.accept) {
        if (c.sum_bins < 128 || c.sum_bins > 1024 * c.B) return set_err(ctx, GB_ERR_INVALID, "store_bins out of range");
        if (!c.logu || !c.accepted_out) return set_err(ctx, GB_ERR_INVALID, "NULL logu / accepted_out");
        if (c.accept == 2) {
            K = (int)(c.B >> 18);   // ~ 2^18 rows per chunk: enough work per launch to hide its tail
            if (K > nw) K = nw;
            if (K > 8) K = 8;       // measured on B200 (config 5): 8 chunks 46.8 ms, 4: 47.1, 16: 47.5 (more launches, more tails)
            if (K < 1) K = 1;
        }

        // large batches: a CTA reserves store slots and list positions a few at a time (one round trip per pool_r accepted
        // rows) and may leave part of its last reservation unused in every launch; small batches reserve exactly
        for (int cN = 0; cN < 4; cN++) {
            const int Nc = 128 << cN;
            pool_r[cN] = c.B >= (1 << 18) ? (cN == 0 ? 8 : cN == 1 ? 4 : 2) : 1;
            const int64_t ctas = (int64_t)ctx->grid_blocks_acc[4 * cN];   // (the general-path kernels reserve one at a time)
            store_slack += ctas * K * (pool_r[cN] - 1) * 2 * Nc;
            ent_slack += ctas * K * (pool_r[cN] - 1);
        }
        if (K > 1 && (2 * c.sum_bins + store_slack) / kPieceElems + 1024 > 0x7fffffff)
            return set_err(ctx, GB_ERR_INVALID, "store_bins too large for the fused update (piece positions are 32-bit)");
        if ((rc = ensure_cap(ctx, &ctx->d_wkeep, &ctx->cap_wkeep, 2 * c.sum_bins + store_slack, true))) return rc;
        if ((rc = ensure_cap(ctx, &ctx->d_wk, &ctx->cap_wk, kWkInts))) return rc;
        if ((rc = ensure_cap(ctx, &ctx->d_ent, &ctx->cap_ent, c.B + ent_slack))) return rc;
        if ((rc = ensure_cap(ctx, &ctx->d_accpar, &ctx->cap_accpar, c.B))) return rc;
        if (K > 1 && (rc = ensure_cap(ctx, &ctx->d_whist, &ctx->cap_whist, nw))) return rc;
        if (K > 1 && (rc = ensure_cap(ctx, &ctx->d_pieces, &ctx->cap_pieces, (2 * c.sum_bins + store_slack) / kPieceElems + 1024))) return rc;
        GB_CUDA(ctx, cudaMemsetAsync(ctx->d_wk, 0, sizeof(int32_t) * kWkInts, st));
    }
    int32_t* chunk_first = ctx->d_wk ? ctx->d_wk + 8 : nullptr;   // zeroed with the counters: one chunk = every walker in chunk 0
    int32_t* bin_count = ctx->d_wk ? ctx->d_wk + kWkHeader : nullptr;
    int32_t* bin_off = bin_count ? bin_count + kNumClasses * kMaxChunks : nullptr;
    int32_t* bin_cursor = bin_count ? bin_count + 2 * kNumClasses * kMaxChunks : nullptr;
    int32_t* bin_ticket = bin_count ? bin_count + 3 * kNumClasses * kMaxChunks : nullptr;

    GB_CUDA(ctx, cudaMemsetAsync(ctx->d_counts, 0, sizeof(int32_t) * 2 * kNumClasses, st));

    PrepArgs p{};
    p.params_new = c.params_new;
    p.params_old = c.params_old;
    p.walker_index = c.walker_index;
    p.move = c.mode == MODE_WAVEFORM ? nullptr : c.move;
    p.accepted = c.accepted;
    p.n_bins = c.n_bins;
    p.move_all = c.mode == MODE_WAVEFORM ? GB_ADD : c.move_all;
    p.N = c.N;
    p.mode = c.mode;
    p.n_walkers = c.data ? c.data->n_walkers : 0;
    p.n_psd = c.data ? c.data->n_psd : 0;
    p.keep = c.keep;
    p.Nmax = c.Nmax;
    p.walker_psd = c.data ? c.data->walker_psd : nullptr;
    p.B = c.B;
    p.Tobs = ctx->cfg.Tobs;
    p.tau = ctx->cfg.armlength / kCLight;
    p.Rmax = ctx->cfg.au / kCLight;
    p.kmax = (int64_t)floor(ctx->cfg.Tobs / (2.0 * ctx->cfg.dt));
    p.src_new = ctx->d_src_new;
    p.src_old = ctx->d_src_old;
    p.lists = ctx->d_lists;
    p.counts = ctx->d_counts;
    p.errflag = ctx->d_counts + 2 * kNumClasses;
    p.dlnL_out = (c.mode == MODE_DLNL || c.mode == MODE_OVERLAP) ? c.dlnL_out : nullptr;
    const unsigned pgrid = (unsigned)((c.B + 255) / 256);
    // binned work lists of gb_delta_loglike_accept.  Up to 2^27 rows: ONE pass -- a bin's list starts where its walker chunk
    // starts among the rows of its class (room for every row of the chunk), its length is the final append cursor.  Beyond
    // that (32-bit list offsets): count the rows of every (class, walker chunk) bin, scan, then the full pass.
    const bool one_pass = c.accept && c.B <= ((int64_t)1 << 27);
    if (c.accept) {
        p.accept = 1;
        p.K = K;
        p.chunk_first = chunk_first;
        if (K > 1) {
            GB_CUDA(ctx, cudaMemsetAsync(ctx->d_whist, 0, sizeof(int32_t) * (size_t)nw, st));
            gb_walker_hist_kernel<<<pgrid, 256, 0, st>>>(c.walker_index, c.B, nw, ctx->d_whist);
            gb_chunk_bounds_kernel<<<1, 1, 0, st>>>(ctx->d_whist, nw, K, c.B, chunk_first, chunk_first + 8);   // (K <= 8)
            ctx->launches += 2;
        }
        p.logq = c.logq;
        p.logu = c.logu;
        p.beta = c.beta;
        p.accpar = ctx->d_accpar;
        p.bin_count = bin_count;
        p.bin_off = bin_off;
        p.bin_cursor = bin_cursor;
        p.accepted_out = c.accepted_out;
        if (one_pass) {
            gb_bin_off_kernel<<<1, kNumClasses * kMaxChunks, 0, st>>>(K > 1 ? chunk_first + 8 : nullptr, c.B, K, bin_off);
            ctx->launches++;
        } else {
            gb_prep_kernel<<<pgrid, 256, 0, st>>>(p);
            gb_bin_scan_kernel<<<1, 1, 0, st>>>(bin_count, bin_off, kNumClasses * K);
            ctx->launches += 2;
        }
        GB_CUDA(ctx, cudaGetLastError());
        p.accept = 2;
    }
    gb_prep_kernel<<<pgrid, 256, 0, st>>>(p);
    ctx->launches++;
    GB_CUDA(ctx, cudaGetLastError());

    MainArgs a{};
    a.src_new = ctx->d_src_new;
    a.src_old = ctx->d_src_old;
    a.lists = ctx->d_lists;
    a.counts = ctx->d_counts;
    a.counters = ctx->d_counts + kNumClasses;
    a.tw = ctx->d_tw;
    a.B = c.B;
    a.mode = c.mode;
    if (c.data) {
        a.resid = c.data->resid;
        a.psd = c.data->psd;
        a.walker_psd = c.data->walker_psd;
        a.k_lo = c.data->k_lo;
        a.n_f = c.data->n_f;
        a.n_walkers = c.data->n_walkers;
        a.n_psd = c.data->n_psd;
        a.psd_is_inverse = c.data->psd_is_inverse;
    }
    a.walker_index = c.walker_index;
    a.move = p.move;
    a.move_all = p.move_all;
    a.dlnL_out = c.dlnL_out;
    a.aux_out = c.aux_out;
    a.AE_out = c.AE_out;
    a.kmin_out = c.kmin_out;
    a.Nmax = c.Nmax;
    a.Tobs = ctx->cfg.Tobs;
    a.tau = p.tau;
    a.wkeep = (c.keep || c.accept) ? ctx->d_wkeep : nullptr;
    a.wkeep_cap = (c.keep || c.accept) ? 2 * c.sum_bins : 0;
    a.errflag = p.errflag;
    if (c.accept) {
        a.ent = ctx->d_ent;
        a.ent_cap = ctx->cap_ent;
        a.wkeep_cap = ctx->cap_wkeep < 2 * c.sum_bins + store_slack ? ctx->cap_wkeep : 2 * c.sum_bins + store_slack;
        a.accpar = ctx->d_accpar;
        a.accepted_out = c.accepted_out;
        a.store_cursor = reinterpret_cast<unsigned long long*>(ctx->d_wk);
        a.ent_cursor = ctx->d_wk + 2;
        a.sc_claim = ctx->d_wk + 3;
        a.n_pieces = ctx->d_wk + 4;
        a.pieces = ctx->d_pieces;
        a.bin_count = one_pass ? bin_cursor : bin_count;
        a.bin_off = bin_off;
        a.bin_ticket = bin_ticket;
        a.K = K;
        a.fuse = c.accept == 2 && K > 1;
        PiecesArgs pa{};
        pa.ent = ctx->d_ent;
        pa.pieces = ctx->d_pieces;
        pa.pieces_cap = ctx->cap_pieces;
        pa.ent_cap = ctx->cap_ent;
        pa.ent_cursor = a.ent_cursor;
        pa.ent_done = ctx->d_wk + 5;
        pa.piece_cursor = ctx->d_wk + 6;
        pa.k_lo = c.data->k_lo;
        pa.n_f = c.data->n_f;
        pa.n_walkers = c.data->n_walkers;
        for (int chunk = 0; chunk < K; chunk++) {
            a.chunk = chunk;
            if (chunk > 0 && a.fuse) {   // the accepted rows of the chunks before this one are complete from here on
                gb_pieces_kernel<<<ctx->num_sms, 256, 0, st>>>(pa);
                gb_ready_kernel<<<1, 1, 0, st>>>(a.ent_cursor, ctx->d_wk + 5, ctx->d_wk + 6, a.sc_claim, ctx->d_wk + 4);
                ctx->launches += 2;
            }
            // the rows outside the fast path first (usually none), then the fast kernels; the classes of a chunk side by side
            // (only when the call is one chunk: with the fused update running, classes side by side measured 47.3 instead of
            // 46.7 ms on config 5 -- the launches of a chunk are then kept in order)
            Fan fan{ctx, st, c.n_bins != nullptr && K == 1, 0};
            if ((rc = fan.begin())) return rc;
            for (int pass = 0; pass < 2; pass++) {
                for (int cN = 3; cN >= 0; cN--) {
                    const int Nc = 128 << cN;
                    if (!c.n_bins && Nc != c.N) continue;
                    a.pool_r = pass ? pool_r[cN] : 1;
                    switch (Nc) {
                        case 128: rc = pass ? launch_main<128, false, true, 1>(ctx, a, c.B, fan.next()) : launch_main<128, false, false, 1>(ctx, a, c.B, fan.next()); break;
                        case 256: rc = pass ? launch_main<256, false, true, 1>(ctx, a, c.B, fan.next()) : launch_main<256, false, false, 1>(ctx, a, c.B, fan.next()); break;
                        case 512: rc = pass ? launch_main<512, false, true, 1>(ctx, a, c.B, fan.next()) : launch_main<512, false, false, 1>(ctx, a, c.B, fan.next()); break;
                        default: rc = pass ? launch_main<1024, false, true, 1>(ctx, a, c.B, fan.next()) : launch_main<1024, false, false, 1>(ctx, a, c.B, fan.next()); break;
                    }
                    if (rc) return rc;
                }
            }
            if ((rc = fan.end())) return rc;
        }
        ctx->kept_B = c.B;
        ctx->kept_cap = a.wkeep_cap;
        ctx->kept_mode = 2;
        if (c.accept == 2) {   // what the fused update left: the pieces nobody took and the last chunk's rows
            if (a.fuse) {
                RestArgs ra{};
                ra.pieces = ctx->d_pieces;
                ra.store = ctx->d_wkeep;
                ra.sc_claim = a.sc_claim;
                ra.n_pieces = ctx->d_wk + 4;
                ra.resid = c.data->resid;
                ra.n_f = c.data->n_f;
                gb_scatter_pieces_kernel<<<ctx->num_sms * 8, 128, 0, st>>>(ra);
                ctx->launches++;
            }
            return scatter_entries(ctx, c.data, 1.0, a.fuse != 0, st);
        }
        if (c.accept == 3) return scatter_entries(ctx, c.data, 1.0, false, st);   // everything, as a separate launch
        return GB_OK;
    }
    // launch only the classes that can occur; largest windows first
    const bool may_swap = c.mode != MODE_WAVEFORM && (c.move ? true : c.move_all == GB_SWAP);   // MODE_OVERLAP: move_all = SWAP
    const bool may_single = c.mode == MODE_WAVEFORM || (c.move ? true : c.move_all != GB_SWAP);
    Fan fan{ctx, st, c.n_bins != nullptr || (may_swap && may_single), 0};
    if ((rc = fan.begin())) return rc;
    for (int cN = 3; cN >= 0; cN--) {
        const int Nc = 128 << cN;
        if (!c.n_bins && Nc != c.N) continue;
        if (may_swap) {
            switch (Nc) {
                case 128: rc = launch_pair<128, true>(ctx, a, c.B, fan); break;
                case 256: rc = launch_pair<256, true>(ctx, a, c.B, fan); break;
                case 512: rc = launch_pair<512, true>(ctx, a, c.B, fan); break;
                default: rc = launch_pair<1024, true>(ctx, a, c.B, fan); break;
            }
            if (rc) return rc;
        }
        if (may_single) {
            switch (Nc) {
                case 128: rc = launch_pair<128, false>(ctx, a, c.B, fan); break;
                case 256: rc = launch_pair<256, false>(ctx, a, c.B, fan); break;
                case 512: rc = launch_pair<512, false>(ctx, a, c.B, fan); break;
                default: rc = launch_pair<1024, false>(ctx, a, c.B, fan); break;
            }
            if (rc) return rc;
        }
    }
    if ((rc = fan.end())) return rc;
    if (c.keep) {
        ctx->kept_B = c.B;
        ctx->kept_cap = 2 * c.sum_bins;
        ctx->kept_mode = 1;
    }
    return GB_OK;
}

}  // namespace

// ------------------------------------------------------------------------------------------------ static scratch
// Scratch of gb_band_sweep_static, the entry point that allocates nothing: a file-scope array in device memory that every
// GPU which loads this library holds until exit.  In HOST code the name g_static_scratch is only a stand-in for the symbol,
// not a device address: a kernel handed &g_static_scratch[0] from the host would fault (or, where the GPU can reach host
// memory, silently use the wrong memory).  The device address is resolved once per device by cudaGetSymbolAddress, with
// that device current (static_scratch_setup, called by gb_create), and that pointer is what the kernels get.
static __device__ __align__(256) unsigned char g_static_scratch[GB_STATIC_SCRATCH_BYTES];

namespace {
constexpr int kMaxDevices = 64;
std::mutex g_static_mu;
void* g_static_ptr[kMaxDevices];   // [device] -> device address of g_static_scratch there (0: not resolved yet)

// requires: cfg.device is the current device
int static_scratch_setup(gb_ctx* ctx) {
    const int d = ctx->cfg.device;
    if (d < 0 || d >= kMaxDevices) return GB_OK;   // such a device gets no static scratch: gb_band_sweep_static says so
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_ptr[d]) {
        void* p = nullptr;
        GB_CUDA(ctx, cudaGetSymbolAddress(&p, g_static_scratch));
        if (!p || (reinterpret_cast<uintptr_t>(p) & 255) != 0)
            return set_err(ctx, GB_ERR_CUDA, "static scratch resolved to a bad address %p on device %d", p, d);
        g_static_ptr[d] = p;
    }
    ctx->d_static = reinterpret_cast<cx*>(g_static_ptr[d]);
    return GB_OK;
}

// gb_band_kernel with the current-source cache of its CTAs in the static array: the grid is one CTA per task (callers
// check n_tasks * N <= GB_STATIC_MAX_TASK_BINS), no allocation, no free
template <int N, bool GEN = false>
int launch_band_static(gb_ctx* ctx, const BandArgs& a, cudaStream_t st) {
    static_assert((size_t)kBandCacheSlots * 2 * sizeof(cx) * GB_STATIC_MAX_TASK_BINS <= (size_t)GB_STATIC_SCRATCH_BYTES,
                  "the static scratch must hold the caches of GB_STATIC_MAX_TASK_BINS / N CTAs");
    const size_t smem = band_smem_bytes<N>(a.max_stage);
    GB_CUDA(ctx, cudaFuncSetAttribute(gb_band_kernel<N, GB_BAND_GM, GEN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int nb = 0;
    GB_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, gb_band_kernel<N, GB_BAND_GM, GEN>, Plan<N>::G * GB_BAND_GM, smem));
    if (nb < 1) return set_err(ctx, GB_ERR_INVALID, "max_stage %d does not fit in shared memory for N = %d", a.max_stage, N);
    int64_t grid = (int64_t)nb * ctx->num_sms;
    if (grid > a.n_tasks) grid = a.n_tasks;
    if ((size_t)grid * kBandCacheSlots * 2 * N * sizeof(cx) > (size_t)GB_STATIC_SCRATCH_BYTES)
        return set_err(ctx, GB_ERR_INVALID, "static scratch too small for %lld CTAs of N = %d", (long long)grid, N);
    BandArgs b = a;
    b.cache = ctx->d_static;
    gb_band_kernel<N, GB_BAND_GM, GEN><<<(unsigned)grid, Plan<N>::G * GB_BAND_GM, smem, st>>>(b);
    ctx->launches++;
    GB_CUDA(ctx, cudaGetLastError());
    return GB_OK;
}
}  // namespace

namespace {
template <int N, bool GEN>
int launch_band(gb_ctx* ctx, const BandArgs& a, cudaStream_t st) {
    const size_t smem = band_smem_bytes<N>(a.max_stage);
    GB_CUDA(ctx, cudaFuncSetAttribute(gb_band_kernel<N, GB_BAND_GM, GEN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int nb = 0;
    GB_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, gb_band_kernel<N, GB_BAND_GM, GEN>, Plan<N>::G * GB_BAND_GM, smem));
    if (nb < 1) return set_err(ctx, GB_ERR_INVALID, "max_stage %d does not fit in shared memory for N = %d", a.max_stage, N);
    int64_t grid = (int64_t)nb * ctx->num_sms;
    if (grid > a.n_tasks) grid = a.n_tasks;
    BandArgs b = a;
    int rc = ensure_cap(ctx, &ctx->d_band_cache, &ctx->cap_band_cache, grid * kBandCacheSlots * 2 * N);
    if (rc) return rc;
    b.cache = ctx->d_band_cache;
    gb_band_kernel<N, GB_BAND_GM, GEN><<<(unsigned)grid, Plan<N>::G * GB_BAND_GM, smem, st>>>(b);
    ctx->launches++;
    GB_CUDA(ctx, cudaGetLastError());
    return GB_OK;
}

template <int N>
int launch_temper(gb_ctx* ctx, const TemperArgs& a, cudaStream_t st) {
    const size_t smem = temper_smem_bytes<N>(a.max_stage);
    GB_CUDA(ctx, cudaFuncSetAttribute(gb_temper_kernel<N, GB_BAND_GM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int nb = 0;
    GB_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, gb_temper_kernel<N, GB_BAND_GM>, Plan<N>::G * GB_BAND_GM, smem));
    if (nb < 1) return set_err(ctx, GB_ERR_INVALID, "max_stage %d does not fit in shared memory for N = %d", a.max_stage, N);
    int64_t grid = (int64_t)nb * ctx->num_sms;
    if (grid > a.n_tasks) grid = a.n_tasks;
    TemperArgs b = a;
    int rc = ensure_cap(ctx, &ctx->d_temper_cache, &ctx->cap_temper_cache, grid * kTemperCacheChains * 2 * a.max_stage);
    if (rc) return rc;
    b.cache = ctx->d_temper_cache;
    gb_temper_kernel<N, GB_BAND_GM><<<(unsigned)grid, Plan<N>::G * GB_BAND_GM, smem, st>>>(b);
    ctx->launches++;
    GB_CUDA(ctx, cudaGetLastError());
    return GB_OK;
}
}  // namespace

// ------------------------------------------------------------------------------------------------ C ABI
extern "C" {

void gb_default_config(gb_config* cfg) {
    if (!cfg) return;
    cfg->Tobs = 31457280.0;
    cfg->dt = 5.0;
    cfg->armlength = 2.5e9;
    cfg->au = 1.495978707e11;
    cfg->year = 31558149.763545603;
    cfg->kappa = 0.0;
    cfg->lambda0 = 0.0;
    cfg->device = 0;
    cfg->reserved = 0;
}

const char* gb_version(void) { return "gbfit-b200 0.1"; }

int gb_create(const gb_config* cfg, gb_ctx** out) {
    if (!cfg || !out) return GB_ERR_INVALID;
    *out = nullptr;
    if (!(cfg->Tobs > 0) || !(cfg->dt > 0) || !(cfg->armlength > 0) || !(cfg->au > 0) || !(cfg->year > 0))
        return GB_ERR_INVALID;
    gb_ctx* ctx = new gb_ctx();
    memset(ctx, 0, sizeof(*ctx));
    ctx->cfg = *cfg;
    *out = ctx;   // returned even on failure so that gb_last_error can be read; caller destroys it
    GB_CUDA(ctx, cudaSetDevice(cfg->device));
    cudaDeviceProp prop;
    GB_CUDA(ctx, cudaGetDeviceProperties(&prop, cfg->device));
    if (prop.major < 10)
        return set_err(ctx, GB_ERR_CUDA, "device %d is sm_%d%d; this library is built for sm_100a only", cfg->device,
                       prop.major, prop.minor);
    ctx->num_sms = prop.multiProcessorCount;
    {
        const int rc_static = static_scratch_setup(ctx);
        if (rc_static) return rc_static;
    }
    OrbitParams op{cfg->Tobs, cfg->armlength, cfg->au, cfg->year, cfg->kappa, cfg->lambda0};
    for (int i = 0; i < 4; i++) {
        const int N = 128 << i;
        std::vector<double> tab((size_t)kOrbitRows * N);
        build_orbit_table(op, N, tab.data());
        GB_CUDA(ctx, cudaMalloc(reinterpret_cast<void**>(&ctx->d_orbit[i]), tab.size() * sizeof(double)));
        GB_CUDA(ctx, cudaMemcpy(ctx->d_orbit[i], tab.data(), tab.size() * sizeof(double), cudaMemcpyHostToDevice));
    }
    std::vector<double> tw(2 * kTwiddleN);
    build_twiddles(tw.data());
    GB_CUDA(ctx, cudaMalloc(reinterpret_cast<void**>(&ctx->d_tw), tw.size() * sizeof(double)));
    GB_CUDA(ctx, cudaMemcpy(ctx->d_tw, tw.data(), tw.size() * sizeof(double), cudaMemcpyHostToDevice));
    GB_CUDA(ctx, cudaMalloc(reinterpret_cast<void**>(&ctx->d_counts), sizeof(int32_t) * (2 * kNumClasses + 1)));
    GB_CUDA(ctx, cudaMemset(ctx->d_counts, 0, sizeof(int32_t) * (2 * kNumClasses + 1)));
    for (int i = 0; i < 3; i++) {
        GB_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->s_side[i], cudaStreamNonBlocking));
        GB_CUDA(ctx, cudaEventCreateWithFlags(&ctx->ev_join[i], cudaEventDisableTiming));
    }
    GB_CUDA(ctx, cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming));
    GB_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->s_in, cudaStreamNonBlocking));
    GB_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->s_out, cudaStreamNonBlocking));
    GB_CUDA(ctx, cudaEventCreateWithFlags(&ctx->ev_start, cudaEventDisableTiming));
    for (int i = 0; i < kHostChunks; i++) {
        GB_CUDA(ctx, cudaEventCreateWithFlags(&ctx->ev_in[i], cudaEventDisableTiming));
        GB_CUDA(ctx, cudaEventCreateWithFlags(&ctx->ev_done[i], cudaEventDisableTiming));
    }
    int rc;
#define GB_SETUP(N_)                                                    \
    if ((rc = setup_kernel<N_, false, true>(ctx))) return rc;           \
    if ((rc = setup_kernel<N_, true, true>(ctx))) return rc;            \
    if ((rc = setup_kernel<N_, false, false>(ctx))) return rc;          \
    if ((rc = setup_kernel<N_, true, false>(ctx))) return rc;           \
    if ((rc = setup_kernel<N_, false, true, 1>(ctx))) return rc;        \
    if ((rc = setup_kernel<N_, false, false, 1>(ctx))) return rc;       \
    if ((rc = setup_kernel<N_, false, true, 2>(ctx))) return rc;
    GB_SETUP(128) GB_SETUP(256) GB_SETUP(512) GB_SETUP(1024)
#undef GB_SETUP
    return GB_OK;
}

void gb_destroy(gb_ctx* ctx) {
    if (!ctx) return;
    cudaSetDevice(ctx->cfg.device);
    cudaDeviceSynchronize();
    for (int i = 0; i < 4; i++) cudaFree(ctx->d_orbit[i]);
    cudaFree(ctx->d_tw);
    cudaFree(ctx->d_counts);
    cudaFree(ctx->d_src_new);
    cudaFree(ctx->d_src_old);
    cudaFree(ctx->d_lists);
    cudaFree(ctx->d_band_cache);
    cudaFree(ctx->d_temper_cache);
    cudaFree(ctx->d_wkeep);
    cudaFree(ctx->d_wk);
    cudaFree(ctx->d_ent);
    cudaFree(ctx->d_accpar);
    cudaFree(ctx->d_pieces);
    cudaFree(ctx->d_whist);
    cudaFree(ctx->d_stage);
    for (int i = 0; i < 3; i++) {
        if (ctx->s_side[i]) cudaStreamDestroy(ctx->s_side[i]);
        if (ctx->ev_join[i]) cudaEventDestroy(ctx->ev_join[i]);
    }
    if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
    if (ctx->s_in) cudaStreamDestroy(ctx->s_in);
    if (ctx->s_out) cudaStreamDestroy(ctx->s_out);
    if (ctx->ev_start) cudaEventDestroy(ctx->ev_start);
    for (int i = 0; i < kHostChunks; i++) {
        if (ctx->ev_in[i]) cudaEventDestroy(ctx->ev_in[i]);
        if (ctx->ev_done[i]) cudaEventDestroy(ctx->ev_done[i]);
    }
    delete ctx;
}

const char* gb_last_error(const gb_ctx* ctx) { return ctx ? ctx->err : "NULL context"; }

int64_t gb_launch_count(const gb_ctx* ctx) { return ctx ? ctx->launches : 0; }

int64_t gb_scratch_bytes(const gb_ctx* ctx) {
    if (!ctx) return 0;
    return ctx->cap_new * (int64_t)sizeof(SrcConst) + ctx->cap_old * (int64_t)sizeof(SrcConst) + ctx->cap_lists * 4 +
           ctx->cap_band_cache * (int64_t)sizeof(cx) + ctx->cap_temper_cache * (int64_t)sizeof(cx) +
           ctx->cap_wkeep * (int64_t)sizeof(cx) + ctx->cap_wk * 4 + ctx->cap_ent * (int64_t)sizeof(KeptEnt) +
           ctx->cap_accpar * (int64_t)sizeof(double4) + ctx->cap_pieces * (int64_t)sizeof(Piece) + ctx->cap_whist * 4 +
           (int64_t)ctx->cap_stage;
}

int gb_measure_fp64_peak(gb_ctx* ctx, double* tflops_out, double* dfma_per_clk_sm_out, double clock_mhz, void* stream) {
    if (!ctx || !tflops_out) return GB_ERR_INVALID;
    GB_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    double* d_sink = nullptr;
    GB_CUDA(ctx, cudaMalloc(reinterpret_cast<void**>(&d_sink), sizeof(double)));
    cudaEvent_t e0, e1;
    GB_CUDA(ctx, cudaEventCreate(&e0));
    GB_CUDA(ctx, cudaEventCreate(&e1));
    const int iters = 8192, threads = 128, grid = ctx->num_sms * 4;
    float best = 0.0f;
    for (int rep = 0; rep < 4; rep++) {   // first repetition warms up
        GB_CUDA(ctx, cudaEventRecord(e0, st));
        gb_dfma_peak_kernel<<<grid, threads, 0, st>>>(d_sink, iters, 1.0000001, 1e-9);
        GB_CUDA(ctx, cudaEventRecord(e1, st));
        GB_CUDA(ctx, cudaEventSynchronize(e1));
        float ms = 0.0f;
        GB_CUDA(ctx, cudaEventElapsedTime(&ms, e0, e1));
        if (rep > 0 && (best == 0.0f || ms < best)) best = ms;
    }
    ctx->launches += 4;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d_sink);
    const double dfma = (double)grid * threads * (double)iters * 8.0 * 8.0;
    *tflops_out = 2.0 * dfma / (best * 1e-3) / 1e12;
    if (dfma_per_clk_sm_out) *dfma_per_clk_sm_out = clock_mhz > 0 ? dfma / (best * 1e-3) / ctx->num_sms / (clock_mhz * 1e6) : 0.0;
    return GB_OK;
}

int gb_check(gb_ctx* ctx, void* stream) {
    if (!ctx) return GB_ERR_INVALID;
    GB_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    int32_t flag = 0;
    GB_CUDA(ctx, cudaMemcpyAsync(&flag, ctx->d_counts + 2 * kNumClasses, sizeof(flag), cudaMemcpyDeviceToHost, st));
    GB_CUDA(ctx, cudaStreamSynchronize(st));
    if (flag) {
        GB_CUDA(ctx, cudaMemsetAsync(ctx->d_counts + 2 * kNumClasses, 0, sizeof(int32_t), st));
        return set_err(ctx, GB_ERR_ROW, "row error flags 0x%x (1: bad N / move / walker index, 2: window beyond Nyquist, 4: sum_n_bins too small)", flag);
    }
    return GB_OK;
}

int gb_waveform(gb_ctx* ctx, const double* params, int64_t B, int N, const int32_t* n_bins, int Nmax, double* AE_out,
                int64_t* kmin_out, void* stream) {
    Call c{};
    c.mode = MODE_WAVEFORM;
    c.params_new = params;
    c.N = N;
    c.n_bins = n_bins;
    c.B = B;
    c.AE_out = AE_out;
    c.kmin_out = kmin_out;
    c.Nmax = Nmax;
    return run_call(ctx, c, stream);
}

int gb_delta_loglike(gb_ctx* ctx, const gb_data* data, const double* params_new, const double* params_old,
                     const int32_t* walker_index, const int8_t* move, int move_all, int N, const int32_t* n_bins,
                     int64_t B, double* dlnL_out, double* aux_out, void* stream) {
    Call c{};
    c.mode = MODE_DLNL;
    c.data = data;
    c.params_new = params_new;
    c.params_old = params_old;
    c.walker_index = walker_index;
    c.move = move;
    c.move_all = move_all;
    c.N = N;
    c.n_bins = n_bins;
    c.B = B;
    c.dlnL_out = dlnL_out;
    c.aux_out = aux_out;
    return run_call(ctx, c, stream);
}

int gb_delta_loglike_keep(gb_ctx* ctx, const gb_data* data, const double* params_new, const double* params_old,
                          const int32_t* walker_index, const int8_t* move, int move_all, int N, const int32_t* n_bins,
                          int64_t B, int64_t sum_n_bins, double* dlnL_out, double* aux_out, void* stream) {
    Call c{};
    c.mode = MODE_DLNL;
    c.data = data;
    c.params_new = params_new;
    c.params_old = params_old;
    c.walker_index = walker_index;
    c.move = move;
    c.move_all = move_all;
    c.N = N;
    c.n_bins = n_bins;
    c.B = B;
    c.dlnL_out = dlnL_out;
    c.aux_out = aux_out;
    c.keep = 1;
    c.sum_bins = n_bins ? sum_n_bins : (int64_t)N * B;
    if (!move && move_all == GB_SWAP) return set_err(ctx, GB_ERR_INVALID, "gb_delta_loglike_keep takes ADD / REMOVE rows only");
    return run_call(ctx, c, stream);
}

int gb_delta_loglike_accept(gb_ctx* ctx, const gb_data* data, const double* params_new, const double* params_old,
                            const int32_t* walker_index, const int8_t* move, int move_all, int N, const int32_t* n_bins,
                            int64_t B, const double* logq, const double* logu, const double* beta, int64_t store_bins,
                            int apply, double* dlnL_out, double* aux_out, uint8_t* accepted_out, void* stream) {
    Call c{};
    c.mode = MODE_DLNL;
    c.data = data;
    c.params_new = params_new;
    c.params_old = params_old;
    c.walker_index = walker_index;
    c.move = move;
    c.move_all = move_all;
    c.N = N;
    c.n_bins = n_bins;
    c.B = B;
    c.dlnL_out = dlnL_out;
    c.aux_out = aux_out;
    c.sum_bins = store_bins;
    c.logq = logq;
    c.logu = logu;
    c.beta = beta;
    c.accepted_out = accepted_out;
    if (apply < 0 || apply > 2) return set_err(ctx, GB_ERR_INVALID, "apply must be 0, 1 or 2");
    c.accept = apply == 0 ? 1 : apply == 1 ? 2 : 3;
    if (!move && move_all == GB_SWAP) return set_err(ctx, GB_ERR_INVALID, "gb_delta_loglike_accept takes ADD / REMOVE rows only");
    return run_call(ctx, c, stream);
}

int gb_residual_update_kept(gb_ctx* ctx, const gb_data* data, const uint8_t* accepted, int negate, void* stream) {
    if (!ctx) return GB_ERR_INVALID;
    if (ctx->kept_B <= 0) return set_err(ctx, GB_ERR_INVALID, "no gb_delta_loglike_keep call to follow");
    if (!data || !data->resid || data->n_f <= 0 || data->n_walkers <= 0) return set_err(ctx, GB_ERR_INVALID, "NULL / empty data view");
    GB_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    if (ctx->kept_mode == 2) {   // after gb_delta_loglike_accept: the accepted rows are the call's own decisions
        if (accepted) return set_err(ctx, GB_ERR_INVALID, "after gb_delta_loglike_accept `accepted` must be NULL (the call decided)");
        return scatter_entries(ctx, data, negate ? -1.0 : 1.0, false, reinterpret_cast<cudaStream_t>(stream));
    }
    KeptArgs a{};
    a.counts = ctx->d_counts;
    a.lists = ctx->d_lists;
    a.src_new = ctx->d_src_new;
    a.src_old = ctx->d_src_old;
    a.wkeep = ctx->d_wkeep;
    a.accepted = accepted;
    a.resid = data->resid;
    a.B = ctx->kept_B;
    a.k_lo = data->k_lo;
    a.n_f = data->n_f;
    a.wkeep_cap = ctx->kept_cap;
    a.n_walkers = data->n_walkers;
    a.errflag = ctx->d_counts + 2 * kNumClasses;
    a.sign = negate ? -1.0 : 1.0;
    gb_scatter_kept_kernel<<<ctx->num_sms * 16, 128, 0, reinterpret_cast<cudaStream_t>(stream)>>>(a);
    ctx->launches++;
    GB_CUDA(ctx, cudaGetLastError());
    return GB_OK;
}

int gb_overlap(gb_ctx* ctx, const gb_data* data, const double* params_a, const double* params_c, const int32_t* psd_row,
               int N, const int32_t* n_bins, int64_t B, double* overlap_out, double* aux_out, void* stream) {
    Call c{};
    c.mode = MODE_OVERLAP;
    c.data = data;
    c.params_new = params_a;
    c.params_old = params_c;
    c.walker_index = psd_row;
    c.move_all = GB_SWAP;
    c.N = N;
    c.n_bins = n_bins;
    c.B = B;
    c.dlnL_out = overlap_out;
    c.aux_out = aux_out;
    return run_call(ctx, c, stream);
}

int gb_residual_update(gb_ctx* ctx, const gb_data* data, const double* params_new, const double* params_old,
                       const int32_t* walker_index, const int8_t* move, int move_all, const uint8_t* accepted, int N,
                       const int32_t* n_bins, int64_t B, void* stream) {
    Call c{};
    c.mode = MODE_UPDATE;
    c.data = data;
    c.params_new = params_new;
    c.params_old = params_old;
    c.walker_index = walker_index;
    c.move = move;
    c.move_all = move_all;
    c.accepted = accepted;
    c.N = N;
    c.n_bins = n_bins;
    c.B = B;
    return run_call(ctx, c, stream);
}

static int band_sweep_call(gb_ctx* ctx, const gb_data* data, const gb_band_task* tasks, int64_t n_tasks, int N, int max_stage,
                           double* params, const int32_t* prop_k, const double* prop_params, const double* prop_logq,
                           const double* prop_logu, const gb_stretch* gen, int32_t* k_out, double* params_out,
                           double* logq_out, double* logu_out, uint8_t* accepted_out, double* dlnL_out, void* stream,
                           bool static_scratch = false) {
    if (!ctx) return GB_ERR_INVALID;
    if (n_tasks < 0 || n_tasks > 0x7fffffff) return set_err(ctx, GB_ERR_INVALID, "n_tasks out of range");
    if (n_tasks == 0) return GB_OK;
    if (!data || !data->resid || !data->psd || data->n_f <= 0 || data->n_walkers <= 0)
        return set_err(ctx, GB_ERR_INVALID, "NULL / empty data view");
    if (!tasks || !params || !accepted_out || !dlnL_out) return set_err(ctx, GB_ERR_INVALID, "NULL argument");
    if (gen) {
        if (!k_out || !params_out || !logq_out || !logu_out) return set_err(ctx, GB_ERR_INVALID, "NULL argument");
        if (!gen->group || gen->n_group < 1 || gen->n_friends < 1 || !(gen->stretch_a > 1.0))
            return set_err(ctx, GB_ERR_INVALID, "bad gb_stretch (group / n_friends / stretch_a)");
        for (int c = 0; c < 8; c++)
            if (!(gen->hi[c] > gen->lo[c])) return set_err(ctx, GB_ERR_INVALID, "bad gb_stretch (prior box)");
    } else if (!prop_k || !prop_params || !prop_logq || !prop_logu) {
        return set_err(ctx, GB_ERR_INVALID, "NULL argument");
    }
    if (!(N == 128 || N == 256 || N == 512 || N == 1024)) return set_err(ctx, GB_ERR_INVALID, "N must be 128, 256, 512 or 1024");
    if (max_stage < 1 || max_stage > GB_BAND_MAX_STAGE) return set_err(ctx, GB_ERR_INVALID, "max_stage out of range");
    GB_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    BandArgs a{};
    a.tasks = tasks;
    a.n_tasks = n_tasks;
    a.params = params;
    a.prop_k = prop_k;
    a.prop_params = prop_params;
    a.prop_logq = prop_logq;
    a.prop_logu = prop_logu;
    if (gen) {
        a.gen = 1;
        a.st = *gen;
        a.gen_k = k_out;
        a.gen_params = params_out;
        a.gen_logq = logq_out;
        a.gen_logu = logu_out;
    }
    a.accepted_out = accepted_out;
    a.dlnL_out = dlnL_out;
    a.orbit = ctx->d_orbit[N == 128 ? 0 : N == 256 ? 1 : N == 512 ? 2 : 3];
    a.tw = ctx->d_tw;
    a.resid = data->resid;
    a.psd = data->psd;
    a.walker_psd = data->walker_psd;
    a.k_lo = data->k_lo;
    a.n_f = data->n_f;
    a.n_walkers = data->n_walkers;
    a.n_psd = data->n_psd;
    a.psd_is_inverse = data->psd_is_inverse;
    a.max_stage = max_stage;
    a.Tobs = ctx->cfg.Tobs;
    a.tau = ctx->cfg.armlength / kCLight;
    a.Rmax = ctx->cfg.au / kCLight;
    a.kmax = (int64_t)floor(ctx->cfg.Tobs / (2.0 * ctx->cfg.dt));
    a.errflag = ctx->d_counts + 2 * kNumClasses;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    if (static_scratch) {
        if (!ctx->d_static)
            return set_err(ctx, GB_ERR_INVALID, "gb_band_sweep_static: no static scratch on device %d (device index >= %d)",
                           ctx->cfg.device, kMaxDevices);
        if (n_tasks * N > GB_STATIC_MAX_TASK_BINS)
            return set_err(ctx, GB_ERR_INVALID,
                           "gb_band_sweep_static: n_tasks * N = %lld exceeds GB_STATIC_MAX_TASK_BINS = %d (the static scratch "
                           "of %d bytes holds the caches of at most %d tasks of N = %d); use gb_band_sweep",
                           (long long)(n_tasks * N), GB_STATIC_MAX_TASK_BINS, GB_STATIC_SCRATCH_BYTES,
                           GB_STATIC_MAX_TASK_BINS / N, N);
        switch (N) {
            case 128: return launch_band_static<128>(ctx, a, st);
            case 256: return launch_band_static<256>(ctx, a, st);
            case 512: return launch_band_static<512>(ctx, a, st);
            default: return launch_band_static<1024>(ctx, a, st);
        }
    }
    if (a.gen) {
        switch (N) {
            case 128: return launch_band<128, true>(ctx, a, st);
            case 256: return launch_band<256, true>(ctx, a, st);
            case 512: return launch_band<512, true>(ctx, a, st);
            default: return launch_band<1024, true>(ctx, a, st);
        }
    }
    switch (N) {
        case 128: return launch_band<128, false>(ctx, a, st);
        case 256: return launch_band<256, false>(ctx, a, st);
        case 512: return launch_band<512, false>(ctx, a, st);
        default: return launch_band<1024, false>(ctx, a, st);
    }
}

int gb_band_sweep(gb_ctx* ctx, const gb_data* data, const gb_band_task* tasks, int64_t n_tasks, int N, int max_stage,
                  double* params, const int32_t* prop_k, const double* prop_params, const double* prop_logq,
                  const double* prop_logu, uint8_t* accepted_out, double* dlnL_out, void* stream) {
    return band_sweep_call(ctx, data, tasks, n_tasks, N, max_stage, params, prop_k, prop_params, prop_logq, prop_logu, nullptr,
                           nullptr, nullptr, nullptr, nullptr, accepted_out, dlnL_out, stream);
}

int gb_band_sweep_static(gb_ctx* ctx, const gb_data* data, const gb_band_task* tasks, int64_t n_tasks, int N, int max_stage,
                         double* params, const int32_t* prop_k, const double* prop_params, const double* prop_logq,
                         const double* prop_logu, uint8_t* accepted_out, double* dlnL_out, void* stream) {
    return band_sweep_call(ctx, data, tasks, n_tasks, N, max_stage, params, prop_k, prop_params, prop_logq, prop_logu, nullptr,
                           nullptr, nullptr, nullptr, nullptr, accepted_out, dlnL_out, stream, true);
}

int gb_band_sweep_generate(gb_ctx* ctx, const gb_data* data, const gb_band_task* tasks, int64_t n_tasks, int N, int max_stage,
                           double* params, const gb_stretch* gen, int32_t* k_out, double* params_out, double* logq_out,
                           double* logu_out, uint8_t* accepted_out, double* dlnL_out, void* stream) {
    if (ctx && !gen) return set_err(ctx, GB_ERR_INVALID, "NULL gb_stretch");
    return band_sweep_call(ctx, data, tasks, n_tasks, N, max_stage, params, nullptr, nullptr, nullptr, nullptr, gen, k_out,
                           params_out, logq_out, logu_out, accepted_out, dlnL_out, stream);
}

int gb_temper_sweep(gb_ctx* ctx, const gb_data* data, const gb_temper_task* tasks, int64_t n_tasks, int N, int max_stage,
                    const double* params, const int32_t* chain_walker, const double* chain_beta,
                    const int32_t* chain_set_begin, const int32_t* chain_set_n, const double* chain_logu,
                    int32_t* perm_out, uint8_t* accepted_out, double* dlnl_out, void* stream) {
    if (!ctx) return GB_ERR_INVALID;
    if (n_tasks < 0 || n_tasks > 0x7fffffff) return set_err(ctx, GB_ERR_INVALID, "n_tasks out of range");
    if (n_tasks == 0) return GB_OK;
    if (!data || !data->resid || !data->psd || data->n_f <= 0 || data->n_walkers <= 0)
        return set_err(ctx, GB_ERR_INVALID, "NULL / empty data view");
    if (!tasks || !params || !chain_walker || !chain_beta || !chain_set_begin || !chain_set_n || !chain_logu || !perm_out ||
        !accepted_out || !dlnl_out)
        return set_err(ctx, GB_ERR_INVALID, "NULL argument");
    if (!(N == 128 || N == 256 || N == 512 || N == 1024)) return set_err(ctx, GB_ERR_INVALID, "N must be 128, 256, 512 or 1024");
    if (max_stage < 1 || max_stage > GB_BAND_MAX_STAGE) return set_err(ctx, GB_ERR_INVALID, "max_stage out of range");
    GB_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    TemperArgs a{};
    a.tasks = tasks;
    a.n_tasks = n_tasks;
    a.params = params;
    a.chain_walker = chain_walker;
    a.chain_beta = chain_beta;
    a.chain_set_begin = chain_set_begin;
    a.chain_set_n = chain_set_n;
    a.chain_logu = chain_logu;
    a.perm_out = perm_out;
    a.accepted_out = accepted_out;
    a.dlnl_out = dlnl_out;
    a.orbit = ctx->d_orbit[N == 128 ? 0 : N == 256 ? 1 : N == 512 ? 2 : 3];
    a.tw = ctx->d_tw;
    a.resid = data->resid;
    a.psd = data->psd;
    a.walker_psd = data->walker_psd;
    a.k_lo = data->k_lo;
    a.n_f = data->n_f;
    a.n_walkers = data->n_walkers;
    a.n_psd = data->n_psd;
    a.psd_is_inverse = data->psd_is_inverse;
    a.max_stage = max_stage;
    a.Tobs = ctx->cfg.Tobs;
    a.tau = ctx->cfg.armlength / kCLight;
    a.Rmax = ctx->cfg.au / kCLight;
    a.kmax = (int64_t)floor(ctx->cfg.Tobs / (2.0 * ctx->cfg.dt));
    a.errflag = ctx->d_counts + 2 * kNumClasses;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    switch (N) {
        case 128: return launch_temper<128>(ctx, a, st);
        case 256: return launch_temper<256>(ctx, a, st);
        case 512: return launch_temper<512>(ctx, a, st);
        default: return launch_temper<1024>(ctx, a, st);
    }
}

}  // extern "C"

// ---- host-buffer forms: one staging buffer, carved per call ----------------------------------------
namespace {
struct Stager {
    gb_ctx* ctx;
    cudaStream_t st;
    char* base;
    size_t off;
    template <typename T>
    T* put(const T* host, size_t count) {   // reserve (and copy in if host != NULL)
        off = (off + 255) & ~(size_t)255;
        T* d = reinterpret_cast<T*>(base + off);
        off += count * sizeof(T);
        if (host) cudaMemcpyAsync(d, host, count * sizeof(T), cudaMemcpyHostToDevice, st);
        return d;
    }
};
int stage_reserve(gb_ctx* ctx, size_t bytes) {
    if (bytes <= ctx->cap_stage) return GB_OK;
    if (ctx->d_stage) {
        GB_CUDA(ctx, cudaDeviceSynchronize());
        GB_CUDA(ctx, cudaFree(ctx->d_stage));
        ctx->d_stage = nullptr;
        ctx->cap_stage = 0;
    }
    if (cudaMalloc(&ctx->d_stage, bytes) != cudaSuccess) {
        cudaGetLastError();
        return set_err(ctx, GB_ERR_NOMEM, "staging allocation of %zu bytes failed", bytes);
    }
    ctx->cap_stage = bytes;
    return GB_OK;
}
}  // namespace

// every error return of a *_host form drains the copy streams first: no copy from or into a caller's host buffer may be in
// flight once the call has returned
namespace {
int drain_on_error(gb_ctx* ctx, void* stream, int rc) {
    if (rc != GB_OK && ctx) {
        const int keep_errno = rc;
        if (ctx->s_in) cudaStreamSynchronize(ctx->s_in);
        if (ctx->s_out) cudaStreamSynchronize(ctx->s_out);
        cudaStreamSynchronize(reinterpret_cast<cudaStream_t>(stream));
        cudaGetLastError();
        return keep_errno;
    }
    return rc;
}

int waveform_host_impl(gb_ctx* ctx, const double* params, int64_t B, int N, const int32_t* n_bins, int Nmax,
                     double* AE_out, int64_t* kmin_out, void* stream) {
    if (!ctx) return GB_ERR_INVALID;
    if (B < 0 || !params || !AE_out || Nmax <= 0) return set_err(ctx, GB_ERR_INVALID, "bad arguments");
    if (B == 0) return GB_OK;
    GB_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    const size_t nAE = (size_t)B * 2 * (size_t)Nmax * 2;
    int rc = stage_reserve(ctx, (size_t)B * (64 + 4 + 8) + nAE * 8 + 4096);
    if (rc) return rc;
    Stager s{ctx, reinterpret_cast<cudaStream_t>(stream), static_cast<char*>(ctx->d_stage), 0};
    double* d_p = s.put(params, (size_t)B * 8);
    int32_t* d_nb = n_bins ? s.put(n_bins, (size_t)B) : nullptr;
    int64_t* d_k = s.put<int64_t>(nullptr, (size_t)B);
    double* d_AE = s.put<double>(nullptr, nAE);
    GB_CUDA(ctx, cudaMemsetAsync(d_AE, 0, nAE * 8, s.st));
    rc = gb_waveform(ctx, d_p, B, N, d_nb, Nmax, d_AE, d_k, stream);
    if (rc) return rc;
    GB_CUDA(ctx, cudaMemcpyAsync(AE_out, d_AE, nAE * 8, cudaMemcpyDeviceToHost, s.st));
    if (kmin_out) GB_CUDA(ctx, cudaMemcpyAsync(kmin_out, d_k, (size_t)B * 8, cudaMemcpyDeviceToHost, s.st));
    GB_CUDA(ctx, cudaStreamSynchronize(s.st));
    return GB_OK;
}

int delta_loglike_host_impl(gb_ctx* ctx, const gb_data* data, const double* params_new, const double* params_old,
                            const int32_t* walker_index, const int8_t* move, int move_all, int N, const int32_t* n_bins,
                            int64_t B, double* dlnL_out, double* aux_out, void* stream) {
    if (!ctx) return GB_ERR_INVALID;
    if (B < 0 || !walker_index || !dlnL_out) return set_err(ctx, GB_ERR_INVALID, "bad arguments");
    if (B == 0) return GB_OK;
    GB_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    int rc = stage_reserve(ctx, (size_t)B * (64 + 64 + 4 + 1 + 4 + 8 + 16) + 8192);
    if (rc) return rc;
    // staging areas for the whole batch; the batch then flows through in chunks: H2D of chunk i+1 (stream s_in) overlaps
    // the kernels of chunk i (caller's stream), whose results go back on s_out
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    Stager s{ctx, st, static_cast<char*>(ctx->d_stage), 0};
    double* d_pn = params_new ? s.put<double>(nullptr, (size_t)B * 8) : nullptr;
    double* d_po = params_old ? s.put<double>(nullptr, (size_t)B * 8) : nullptr;
    int32_t* d_w = s.put<int32_t>(nullptr, (size_t)B);
    int8_t* d_mv = move ? s.put<int8_t>(nullptr, (size_t)B) : nullptr;
    int32_t* d_nb = n_bins ? s.put<int32_t>(nullptr, (size_t)B) : nullptr;
    double* d_out = s.put<double>(nullptr, (size_t)B);
    double* d_aux = aux_out ? s.put<double>(nullptr, (size_t)B * 2) : nullptr;
    const int nch = B >= (1 << 18) ? kHostChunks : 1;
    GB_CUDA(ctx, cudaEventRecord(ctx->ev_start, st));
    GB_CUDA(ctx, cudaStreamWaitEvent(ctx->s_in, ctx->ev_start, 0));   // earlier work on `stream` may still read the staging area
    for (int c = 0; c < nch; c++) {
        const int64_t lo = B * c / nch, n = B * (c + 1) / nch - lo;
        if (d_pn) GB_CUDA(ctx, cudaMemcpyAsync(d_pn + 8 * lo, params_new + 8 * lo, (size_t)n * 64, cudaMemcpyHostToDevice, ctx->s_in));
        if (d_po) GB_CUDA(ctx, cudaMemcpyAsync(d_po + 8 * lo, params_old + 8 * lo, (size_t)n * 64, cudaMemcpyHostToDevice, ctx->s_in));
        GB_CUDA(ctx, cudaMemcpyAsync(d_w + lo, walker_index + lo, (size_t)n * 4, cudaMemcpyHostToDevice, ctx->s_in));
        if (d_mv) GB_CUDA(ctx, cudaMemcpyAsync(d_mv + lo, move + lo, (size_t)n, cudaMemcpyHostToDevice, ctx->s_in));
        if (d_nb) GB_CUDA(ctx, cudaMemcpyAsync(d_nb + lo, n_bins + lo, (size_t)n * 4, cudaMemcpyHostToDevice, ctx->s_in));
        GB_CUDA(ctx, cudaEventRecord(ctx->ev_in[c], ctx->s_in));
    }
    for (int c = 0; c < nch; c++) {
        const int64_t lo = B * c / nch, n = B * (c + 1) / nch - lo;
        GB_CUDA(ctx, cudaStreamWaitEvent(st, ctx->ev_in[c], 0));
        rc = gb_delta_loglike(ctx, data, d_pn ? d_pn + 8 * lo : nullptr, d_po ? d_po + 8 * lo : nullptr, d_w + lo,
                              d_mv ? d_mv + lo : nullptr, move_all, N, d_nb ? d_nb + lo : nullptr, n, d_out + lo,
                              d_aux ? d_aux + 2 * lo : nullptr, stream);
        if (rc) return rc;
        GB_CUDA(ctx, cudaEventRecord(ctx->ev_done[c], st));
        GB_CUDA(ctx, cudaStreamWaitEvent(ctx->s_out, ctx->ev_done[c], 0));
        GB_CUDA(ctx, cudaMemcpyAsync(dlnL_out + lo, d_out + lo, (size_t)n * 8, cudaMemcpyDeviceToHost, ctx->s_out));
        if (aux_out) GB_CUDA(ctx, cudaMemcpyAsync(aux_out + 2 * lo, d_aux + 2 * lo, (size_t)n * 16, cudaMemcpyDeviceToHost, ctx->s_out));
    }
    GB_CUDA(ctx, cudaStreamSynchronize(ctx->s_out));
    GB_CUDA(ctx, cudaStreamSynchronize(st));
    return GB_OK;
}

int delta_loglike_accept_host_impl(gb_ctx* ctx, const gb_data* data, const double* params_new, const double* params_old,
                                   const int32_t* walker_index, const int8_t* move, int move_all, int N, const int32_t* n_bins,
                                   int64_t B, const double* logq, const double* logu, const double* beta, int64_t store_bins,
                                   int apply, double* dlnL_out, double* aux_out, uint8_t* accepted_out, void* stream) {
    if (!ctx) return GB_ERR_INVALID;
    if (B < 0 || !walker_index || !dlnL_out || !logu || !accepted_out) return set_err(ctx, GB_ERR_INVALID, "bad arguments");
    if (B == 0) return GB_OK;
    GB_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    int rc = stage_reserve(ctx, (size_t)B * (64 + 64 + 4 + 1 + 4 + 24 + 8 + 16 + 1) + 16384);
    if (rc) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    Stager s{ctx, st, static_cast<char*>(ctx->d_stage), 0};
    double* d_pn = params_new ? s.put<double>(nullptr, (size_t)B * 8) : nullptr;
    double* d_po = params_old ? s.put<double>(nullptr, (size_t)B * 8) : nullptr;
    int32_t* d_w = s.put<int32_t>(nullptr, (size_t)B);
    int8_t* d_mv = move ? s.put<int8_t>(nullptr, (size_t)B) : nullptr;
    int32_t* d_nb = n_bins ? s.put<int32_t>(nullptr, (size_t)B) : nullptr;
    double* d_lq = logq ? s.put<double>(nullptr, (size_t)B) : nullptr;
    double* d_lu = s.put<double>(nullptr, (size_t)B);
    double* d_bt = beta ? s.put<double>(nullptr, (size_t)B) : nullptr;
    double* d_out = s.put<double>(nullptr, (size_t)B);
    double* d_aux = aux_out ? s.put<double>(nullptr, (size_t)B * 2) : nullptr;
    uint8_t* d_acc = s.put<uint8_t>(nullptr, (size_t)B);
    // chunked as gb_delta_loglike_host; a chunk's update has finished when its last kernel ends, so the next chunk reuses
    // the store.  apply = 0 keeps the state of ONE call for gb_residual_update_kept: a single chunk then
    const int nch = (B >= (1 << 18) && apply != 0) ? kHostChunksAccept : 1;
    // the first chunk is the small one: its copy is the only one no kernel hides (cuts at 2/24, 9/24, 16/24 of the rows)
    static_assert(kHostChunksAccept == 4, "chunk cuts below");
    const int cut24[kHostChunksAccept + 1] = GB_HOST_ACCEPT_CUTS;
    auto cut = [&](int c) -> int64_t { return nch == 1 ? (c ? B : 0) : B * cut24[c] / 24; };
    GB_CUDA(ctx, cudaEventRecord(ctx->ev_start, st));
    GB_CUDA(ctx, cudaStreamWaitEvent(ctx->s_in, ctx->ev_start, 0));
    for (int c = 0; c < nch; c++) {
        const int64_t lo = cut(c), n = cut(c + 1) - lo;
        if (d_pn) GB_CUDA(ctx, cudaMemcpyAsync(d_pn + 8 * lo, params_new + 8 * lo, (size_t)n * 64, cudaMemcpyHostToDevice, ctx->s_in));
        if (d_po) GB_CUDA(ctx, cudaMemcpyAsync(d_po + 8 * lo, params_old + 8 * lo, (size_t)n * 64, cudaMemcpyHostToDevice, ctx->s_in));
        GB_CUDA(ctx, cudaMemcpyAsync(d_w + lo, walker_index + lo, (size_t)n * 4, cudaMemcpyHostToDevice, ctx->s_in));
        if (d_mv) GB_CUDA(ctx, cudaMemcpyAsync(d_mv + lo, move + lo, (size_t)n, cudaMemcpyHostToDevice, ctx->s_in));
        if (d_nb) GB_CUDA(ctx, cudaMemcpyAsync(d_nb + lo, n_bins + lo, (size_t)n * 4, cudaMemcpyHostToDevice, ctx->s_in));
        if (d_lq) GB_CUDA(ctx, cudaMemcpyAsync(d_lq + lo, logq + lo, (size_t)n * 8, cudaMemcpyHostToDevice, ctx->s_in));
        GB_CUDA(ctx, cudaMemcpyAsync(d_lu + lo, logu + lo, (size_t)n * 8, cudaMemcpyHostToDevice, ctx->s_in));
        if (d_bt) GB_CUDA(ctx, cudaMemcpyAsync(d_bt + lo, beta + lo, (size_t)n * 8, cudaMemcpyHostToDevice, ctx->s_in));
        GB_CUDA(ctx, cudaEventRecord(ctx->ev_in[c], ctx->s_in));
    }
    for (int c = 0; c < nch; c++) {
        const int64_t lo = cut(c), n = cut(c + 1) - lo;
        GB_CUDA(ctx, cudaStreamWaitEvent(st, ctx->ev_in[c], 0));
        rc = gb_delta_loglike_accept(ctx, data, d_pn ? d_pn + 8 * lo : nullptr, d_po ? d_po + 8 * lo : nullptr, d_w + lo,
                                     d_mv ? d_mv + lo : nullptr, move_all, N, d_nb ? d_nb + lo : nullptr, n,
                                     d_lq ? d_lq + lo : nullptr, d_lu + lo, d_bt ? d_bt + lo : nullptr,
                                     store_bins < 1024 * n ? store_bins : 1024 * n, apply, d_out + lo,
                                     d_aux ? d_aux + 2 * lo : nullptr, d_acc + lo, stream);
        if (rc) return rc;
        GB_CUDA(ctx, cudaEventRecord(ctx->ev_done[c], st));
        GB_CUDA(ctx, cudaStreamWaitEvent(ctx->s_out, ctx->ev_done[c], 0));
        GB_CUDA(ctx, cudaMemcpyAsync(dlnL_out + lo, d_out + lo, (size_t)n * 8, cudaMemcpyDeviceToHost, ctx->s_out));
        GB_CUDA(ctx, cudaMemcpyAsync(accepted_out + lo, d_acc + lo, (size_t)n, cudaMemcpyDeviceToHost, ctx->s_out));
        if (aux_out) GB_CUDA(ctx, cudaMemcpyAsync(aux_out + 2 * lo, d_aux + 2 * lo, (size_t)n * 16, cudaMemcpyDeviceToHost, ctx->s_out));
    }
    GB_CUDA(ctx, cudaStreamSynchronize(ctx->s_out));
    GB_CUDA(ctx, cudaStreamSynchronize(st));
    return GB_OK;
}

int residual_update_host_impl(gb_ctx* ctx, const gb_data* data, const double* params_new, const double* params_old,
                              const int32_t* walker_index, const int8_t* move, int move_all, const uint8_t* accepted,
                              int N, const int32_t* n_bins, int64_t B, void* stream) {
    if (!ctx) return GB_ERR_INVALID;
    if (B < 0 || !walker_index) return set_err(ctx, GB_ERR_INVALID, "bad arguments");
    if (B == 0) return GB_OK;
    GB_CUDA(ctx, cudaSetDevice(ctx->cfg.device));
    int rc = stage_reserve(ctx, (size_t)B * (64 + 64 + 4 + 1 + 1 + 4) + 8192);
    if (rc) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    Stager s{ctx, st, static_cast<char*>(ctx->d_stage), 0};
    double* d_pn = params_new ? s.put<double>(nullptr, (size_t)B * 8) : nullptr;
    double* d_po = params_old ? s.put<double>(nullptr, (size_t)B * 8) : nullptr;
    int32_t* d_w = s.put<int32_t>(nullptr, (size_t)B);
    int8_t* d_mv = move ? s.put<int8_t>(nullptr, (size_t)B) : nullptr;
    uint8_t* d_acc = accepted ? s.put<uint8_t>(nullptr, (size_t)B) : nullptr;
    int32_t* d_nb = n_bins ? s.put<int32_t>(nullptr, (size_t)B) : nullptr;
    const int nch = B >= (1 << 18) ? kHostChunks : 1;   // chunked as gb_delta_loglike_host
    GB_CUDA(ctx, cudaEventRecord(ctx->ev_start, st));
    GB_CUDA(ctx, cudaStreamWaitEvent(ctx->s_in, ctx->ev_start, 0));
    for (int c = 0; c < nch; c++) {
        const int64_t lo = B * c / nch, n = B * (c + 1) / nch - lo;
        if (d_acc) GB_CUDA(ctx, cudaMemcpyAsync(d_acc + lo, accepted + lo, (size_t)n, cudaMemcpyHostToDevice, ctx->s_in));
        if (d_pn) GB_CUDA(ctx, cudaMemcpyAsync(d_pn + 8 * lo, params_new + 8 * lo, (size_t)n * 64, cudaMemcpyHostToDevice, ctx->s_in));
        if (d_po) GB_CUDA(ctx, cudaMemcpyAsync(d_po + 8 * lo, params_old + 8 * lo, (size_t)n * 64, cudaMemcpyHostToDevice, ctx->s_in));
        GB_CUDA(ctx, cudaMemcpyAsync(d_w + lo, walker_index + lo, (size_t)n * 4, cudaMemcpyHostToDevice, ctx->s_in));
        if (d_mv) GB_CUDA(ctx, cudaMemcpyAsync(d_mv + lo, move + lo, (size_t)n, cudaMemcpyHostToDevice, ctx->s_in));
        if (d_nb) GB_CUDA(ctx, cudaMemcpyAsync(d_nb + lo, n_bins + lo, (size_t)n * 4, cudaMemcpyHostToDevice, ctx->s_in));
        GB_CUDA(ctx, cudaEventRecord(ctx->ev_in[c], ctx->s_in));
    }
    for (int c = 0; c < nch; c++) {
        const int64_t lo = B * c / nch, n = B * (c + 1) / nch - lo;
        GB_CUDA(ctx, cudaStreamWaitEvent(st, ctx->ev_in[c], 0));
        rc = gb_residual_update(ctx, data, d_pn ? d_pn + 8 * lo : nullptr, d_po ? d_po + 8 * lo : nullptr, d_w + lo,
                                d_mv ? d_mv + lo : nullptr, move_all, d_acc ? d_acc + lo : nullptr, N,
                                d_nb ? d_nb + lo : nullptr, n, stream);
        if (rc) return rc;
    }
    GB_CUDA(ctx, cudaStreamSynchronize(st));
    return GB_OK;
}
}  // namespace

extern "C" {

int gb_waveform_host(gb_ctx* ctx, const double* params, int64_t B, int N, const int32_t* n_bins, int Nmax,
                     double* AE_out, int64_t* kmin_out, void* stream) {
    return drain_on_error(ctx, stream, waveform_host_impl(ctx, params, B, N, n_bins, Nmax, AE_out, kmin_out, stream));
}

int gb_delta_loglike_host(gb_ctx* ctx, const gb_data* data, const double* params_new, const double* params_old,
                          const int32_t* walker_index, const int8_t* move, int move_all, int N, const int32_t* n_bins,
                          int64_t B, double* dlnL_out, double* aux_out, void* stream) {
    return drain_on_error(ctx, stream, delta_loglike_host_impl(ctx, data, params_new, params_old, walker_index, move, move_all,
                                                               N, n_bins, B, dlnL_out, aux_out, stream));
}

int gb_delta_loglike_accept_host(gb_ctx* ctx, const gb_data* data, const double* params_new, const double* params_old,
                                 const int32_t* walker_index, const int8_t* move, int move_all, int N, const int32_t* n_bins,
                                 int64_t B, const double* logq, const double* logu, const double* beta, int64_t store_bins,
                                 int apply, double* dlnL_out, double* aux_out, uint8_t* accepted_out, void* stream) {
    return drain_on_error(ctx, stream, delta_loglike_accept_host_impl(ctx, data, params_new, params_old, walker_index, move,
                                                                      move_all, N, n_bins, B, logq, logu, beta, store_bins,
                                                                      apply, dlnL_out, aux_out, accepted_out, stream));
}

int gb_residual_update_host(gb_ctx* ctx, const gb_data* data, const double* params_new, const double* params_old,
                            const int32_t* walker_index, const int8_t* move, int move_all, const uint8_t* accepted,
                            int N, const int32_t* n_bins, int64_t B, void* stream) {
    return drain_on_error(ctx, stream, residual_update_host_impl(ctx, data, params_new, params_old, walker_index, move,
                                                                 move_all, accepted, N, n_bins, B, stream));
}

}  // extern "C"
