// gb_fft.cuh -- length-N complex128 FFT held entirely in shared memory (step O6 of DESIGN.md).
//
// Stockham-style mixed-radix decimation in time, executed in place by a group of G threads:
// every stage each thread reads R inputs at stride N/R (conflict-free: consecutive threads, consecutive
// 16-byte elements), the group synchronises, the thread applies its twiddles and an R-point DFT in
// registers and writes the R outputs at stride Ns, and the group synchronises again.  The first stage's
// strided writes would be 8-way bank conflicted; one pad element after every 8 removes the conflict
// (pad(a) = a + a/8).  Output is in natural order.  Both channels (A, E) share the twiddle loads.
//
// The per-thread halves (read / compute+write) are plain __host__ __device__ functions so that the host
// logic test can replay a stage thread by thread; the barriers live in the kernels (gbfit.cu).
#pragma once
#include "gb_math.cuh"

namespace gbk {

struct alignas(16) cx {   // complex128 element of the shared-memory buffers (layout of double2)
    double re, im;
};

GB_HD constexpr int pad_idx(int a) { return a + (a >> 3); }
GB_HD constexpr int padded_len(int N) { return N + (N >> 3); }

GB_HD void bf(cx& a, cx& b) {
    const cx t = a;
    a = {t.re + b.re, t.im + b.im};
    b = {t.re - b.re, t.im - b.im};
}
GB_HD cx mul_mi(cx a) { return {a.im, -a.re}; }                 // a * (-i)
GB_HD cx cxmul(cx a, cx w) { return {a.re * w.re - a.im * w.im, a.re * w.im + a.im * w.re}; }

// In-register forward DFTs (sign exp(-2 pi i jk/R)), decimation in frequency.  On return v[] holds the
// outputs in bit-reversed order: output r is v[bitrev_R(r)].
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

template <int R>
GB_HD constexpr int bitrev(int r) {
    int out = 0;
    for (int b = 1, m = R >> 1; b < R; b <<= 1, m >>= 1)
        if (r & b) out |= m;
    return out;
}

// One stage, per-thread register state: PER butterflies of R points for both channels.
template <int N, int G, int R>
struct StageRegs {
    static constexpr int NB = N / R;
    static constexpr int PER = NB / G;
    static_assert(PER >= 1 && PER * G == NB, "group size must divide the butterfly count");
    cx a[PER][R], e[PER][R];
};

template <int N, int G, int R>
GB_HD void fft_stage_read(const cx* bA, const cx* bE, int tid, StageRegs<N, G, R>& rg) {
    constexpr int NB = N / R, PER = NB / G;
#pragma unroll
    for (int p = 0; p < PER; p++) {
        const int j = tid + p * G;
#pragma unroll
        for (int r = 0; r < R; r++) {
            rg.a[p][r] = bA[pad_idx(j + r * NB)];
            rg.e[p][r] = bE[pad_idx(j + r * NB)];
        }
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

// tw[k] = exp(-2 pi i k / 1024)
template <int N, int G, int R, int Ns>
GB_HD void fft_stage_write(cx* bA, cx* bE, const cx* tw, int tid, StageRegs<N, G, R>& rg) {
    constexpr int NB = N / R, PER = NB / G;
#pragma unroll
    for (int p = 0; p < PER; p++) {
        const int j = tid + p * G;
        const int k = j & (Ns - 1);
        if (Ns > 1) {
#pragma unroll
            for (int r = 1; r < R; r++) {
                const cx w = GB_LDG_CX(tw + (r * k) * (1024 / (Ns * R)));
                rg.a[p][r] = cxmul(rg.a[p][r], w);
                rg.e[p][r] = cxmul(rg.e[p][r], w);
            }
        }
        dft_regs<R>(rg.a[p]);
        dft_regs<R>(rg.e[p]);
        const int j0 = (j - k) * R + k;
#pragma unroll
        for (int r = 0; r < R; r++) {
            bA[pad_idx(j0 + r * Ns)] = rg.a[p][bitrev<R>(r)];
            bE[pad_idx(j0 + r * Ns)] = rg.e[p][bitrev<R>(r)];
        }
    }
}

// Radix plans (group size G, then the stages as X(N, G, radix, Ns) with Ns = product of the earlier radices):
//   N = 128: 4,4,4,2   256: 8,8,4   512: 8,8,8   1024: 8,8,4,4
// The kernels expand X into read / barrier / write / barrier; the host logic test replays the same list.
template <int N> struct Plan;
template <> struct Plan<128>  { static constexpr int G = 32; };
template <> struct Plan<256>  { static constexpr int G = 32; };
template <> struct Plan<512>  { static constexpr int G = 64; };
template <> struct Plan<1024> { static constexpr int G = 128; };
#define GB_FFT_PLAN_128(X)  X(128, 32, 4, 1) X(128, 32, 4, 4) X(128, 32, 4, 16) X(128, 32, 2, 64)
#define GB_FFT_PLAN_256(X)  X(256, 32, 8, 1) X(256, 32, 8, 8) X(256, 32, 4, 64)
#define GB_FFT_PLAN_512(X)  X(512, 64, 8, 1) X(512, 64, 8, 8) X(512, 64, 8, 64)
#define GB_FFT_PLAN_1024(X) X(1024, 128, 8, 1) X(1024, 128, 8, 8) X(1024, 128, 4, 64) X(1024, 128, 4, 256)

}  // namespace gbk
