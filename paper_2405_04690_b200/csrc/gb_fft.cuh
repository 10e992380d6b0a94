// gb_fft.cuh -- length-N complex128 FFT held entirely in shared memory (step O6 of DESIGN.md).
//
// The FFT of this path is bound by shared-memory bandwidth (16-byte elements, 128 B/clk per SM), not by its
// flops, so the design minimises round trips through shared memory:
//   * Stockham-style mixed-radix decimation in time with HIGH radices (16 / 8 / 4): 2 stages for N = 256,
//     3 for N = 128, 512, 1024;
//   * the two channels are split over the group: threads [0, H) of the G = 2H threads transform A, threads
//     [H, 2H) transform E, so one thread holds up to 16 complex points of ONE channel in registers;
//   * every stage each thread reads R inputs at stride N/R (consecutive threads, consecutive 16-byte
//     elements: conflict-free), applies its twiddles and an R-point DFT in registers, and writes R outputs at
//     stride Ns; the first stage's strided writes are kept conflict-free by one pad element after every 8
//     (first radix 8) or 16 (first radix 16) elements;
//   * the LAST stage is not written back: its outputs stay in registers, where thread ht of a channel holds
//     the bins j = ht + H m, m = 0 .. N/H - 1 -- consecutive threads, consecutive bins -- so the epilogue
//     (waveform store, inner products, scatter) reads them directly with coalesced global accesses.
//     (The SWAP kernels, which need both waveforms side by side, write the last stage back instead.)
// Output is in natural order.  Twiddles come from one table tw[k] = exp(-2 pi i k / 1024).
//
// The per-thread pieces are plain __host__ __device__ functions so that the host logic test can replay a
// stage thread by thread; the barriers live in the kernels (gbfit.cu).
#pragma once
#include "gb_math.cuh"

namespace gbk {

struct alignas(16) cx {   // complex128 element of the shared-memory buffers (layout of double2)
    double re, im;
};

// Group size G (threads per item), and log2 of the padding period.  Stage lists: X(N, R, Ns) for the stages
// that are written back, L(N, R, Ns) for the last one; Ns = product of the earlier radices.
template <int N> struct Plan;
template <> struct Plan<128>  { static constexpr int G = 32,  PADSH = 3; };
template <> struct Plan<256>  { static constexpr int G = 32,  PADSH = 4; };
template <> struct Plan<512>  { static constexpr int G = 64,  PADSH = 3; };
template <> struct Plan<1024> { static constexpr int G = 128, PADSH = 4; };
#define GB_FFT_PLAN_128(X, L)  X(128, 8, 1)   X(128, 4, 8)    L(128, 4, 32)
#define GB_FFT_PLAN_256(X, L)  X(256, 16, 1)  L(256, 16, 16)
#define GB_FFT_PLAN_512(X, L)  X(512, 8, 1)   X(512, 8, 8)    L(512, 8, 64)
#define GB_FFT_PLAN_1024(X, L) X(1024, 16, 1) X(1024, 16, 16) L(1024, 4, 256)

template <int N> GB_HD constexpr int pad_idx(int a) { return a + (a >> Plan<N>::PADSH); }
template <int N> GB_HD constexpr int padded_len() { return N + (N >> Plan<N>::PADSH); }

GB_HD void bf(cx& a, cx& b) {
    const cx t = a;
    a = {t.re + b.re, t.im + b.im};
    b = {t.re - b.re, t.im - b.im};
}
GB_HD cx mul_mi(cx a) { return {a.im, -a.re}; }                 // a * (-i)
GB_HD cx cxmul(cx a, cx w) { return {a.re * w.re - a.im * w.im, a.re * w.im + a.im * w.re}; }

// In-register forward DFTs (sign exp(-2 pi i jk/R)), decimation in frequency.  On return v[] holds the
// outputs in bit-reversed order: output r is v[bitrev<R>(r)].
template <int R>
GB_HD void dft_regs(cx* v);

template <>
GB_HD void dft_regs<2>(cx* v) {
    bf(v[0], v[1]);
}
template <>
GB_HD void dft_regs<4>(cx* v) {
    bf(v[0], v[2]);
    bf(v[1], v[3]);
    v[3] = mul_mi(v[3]);
    bf(v[0], v[1]);
    bf(v[2], v[3]);
}
template <>
GB_HD void dft_regs<8>(cx* v) {
    constexpr double h = 0.70710678118654752440;
    bf(v[0], v[4]);
    bf(v[1], v[5]);
    bf(v[2], v[6]);
    bf(v[3], v[7]);
    v[5] = {(v[5].re + v[5].im) * h, (v[5].im - v[5].re) * h};   // * W8
    v[6] = mul_mi(v[6]);                                         // * W8^2
    v[7] = {(v[7].im - v[7].re) * h, -(v[7].re + v[7].im) * h};  // * W8^3
    bf(v[0], v[2]);
    bf(v[1], v[3]);
    bf(v[4], v[6]);
    bf(v[5], v[7]);
    v[3] = mul_mi(v[3]);
    v[7] = mul_mi(v[7]);
    bf(v[0], v[1]);
    bf(v[2], v[3]);
    bf(v[4], v[5]);
    bf(v[6], v[7]);
}
template <>
GB_HD void dft_regs<16>(cx* v) {
    constexpr double h = 0.70710678118654752440;    // cos(pi/4)
    constexpr double c1 = 0.92387953251128675613;   // cos(pi/8)
    constexpr double s1 = 0.38268343236508977173;   // sin(pi/8)
#pragma unroll
    for (int i = 0; i < 8; i++) bf(v[i], v[i + 8]);
    // second half times W16^i = exp(-2 pi i * i / 16), i = 0..7; then an 8-point DFT of each half
    v[9] = cxmul(v[9], {c1, -s1});
    v[10] = {(v[10].re + v[10].im) * h, (v[10].im - v[10].re) * h};
    v[11] = cxmul(v[11], {s1, -c1});
    v[12] = mul_mi(v[12]);
    v[13] = cxmul(v[13], {-s1, -c1});
    v[14] = {(v[14].im - v[14].re) * h, -(v[14].re + v[14].im) * h};
    v[15] = cxmul(v[15], {-c1, -s1});
    dft_regs<8>(v);
    dft_regs<8>(v + 8);
}

template <int R>
GB_HD constexpr int bitrev(int r) {
    int out = 0;
    for (int b = 1, m = R >> 1; b < R; b <<= 1, m >>= 1)
        if (r & b) out |= m;
    return out;
}

// One stage of one channel, per-thread register state: PER butterflies of R points.
template <int N, int R>
struct StageRegs {
    static constexpr int H = Plan<N>::G / 2;     // threads per channel
    static constexpr int NB = N / R;             // butterflies per channel
    static constexpr int PER = NB / H;           // butterflies per thread
    static_assert(PER >= 1 && PER * H == NB, "threads per channel must divide the butterfly count");
    cx v[PER][R];
};

// ht = thread index within the channel (0 .. H-1); buf = that channel's padded buffer
template <int N, int R>
GB_HD void fft_stage_read(const cx* buf, int ht, StageRegs<N, R>& rg) {
    constexpr int H = StageRegs<N, R>::H, NB = StageRegs<N, R>::NB, PER = StageRegs<N, R>::PER;
#pragma unroll
    for (int p = 0; p < PER; p++) {
        const int j = ht + p * H;
#pragma unroll
        for (int r = 0; r < R; r++) rg.v[p][r] = buf[pad_idx<N>(j + r * NB)];
    }
}

#if defined(__CUDA_ARCH__)
#define GB_LDG_CX(ptr) gbk::ldg_cx(ptr)
__device__ __forceinline__ cx ldg_cx(const cx* p) {
    const double2 v = __ldg(reinterpret_cast<const double2*>(p));
    return {v.x, v.y};
}
#else
#define GB_LDG_CX(ptr) (*(ptr))
#endif

// twiddles (tw[k] = exp(-2 pi i k / 1024)) and the R-point DFTs, in registers
template <int N, int R, int Ns>
GB_HD void fft_stage_compute(const cx* tw, int ht, StageRegs<N, R>& rg) {
    constexpr int H = StageRegs<N, R>::H, PER = StageRegs<N, R>::PER;
#pragma unroll
    for (int p = 0; p < PER; p++) {
        const int j = ht + p * H;
        const int k = j & (Ns - 1);
        if (Ns > 1) {
#pragma unroll
            for (int r = 1; r < R; r++) rg.v[p][r] = cxmul(rg.v[p][r], GB_LDG_CX(tw + (r * k) * (1024 / (Ns * R))));
        }
        dft_regs<R>(rg.v[p]);
    }
}

// outputs back to the buffer in natural order
template <int N, int R, int Ns>
GB_HD void fft_stage_store(cx* buf, int ht, const StageRegs<N, R>& rg) {
    constexpr int H = StageRegs<N, R>::H, PER = StageRegs<N, R>::PER;
#pragma unroll
    for (int p = 0; p < PER; p++) {
        const int j = ht + p * H;
        const int k = j & (Ns - 1);
        const int j0 = (j - k) * R + k;
#pragma unroll
        for (int r = 0; r < R; r++) buf[pad_idx<N>(j0 + r * Ns)] = rg.v[p][bitrev<R>(r)];
    }
}

// Last stage (Ns * R == N): output bin j = ht + H m, m = 0 .. N/H - 1, is element (m % PER, bitrev(m / PER)).
template <int N, int R>
GB_HD void fft_last_to_bins(const StageRegs<N, R>& rg, cx* h /* [N / H] */) {
    constexpr int PER = StageRegs<N, R>::PER;
#pragma unroll
    for (int r = 0; r < R; r++) {
#pragma unroll
        for (int p = 0; p < PER; p++) h[p + PER * r] = rg.v[p][bitrev<R>(r)];
    }
}

}  // namespace gbk
