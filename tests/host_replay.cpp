// host_replay.cpp -- test-only replay, on the CPU, of the arithmetic the CUDA kernels run (host logic test).
//
// The per-sample functions (gb_math.cuh, gb_fast.cuh) and the per-thread FFT stage halves (gb_fft.cuh) are
// __host__ __device__; this file calls them in the order gb_main_kernel does -- "thread" by "thread", with a
// loop where the kernel has a barrier -- so that the restructured arithmetic of the product path can be
// compared with the oracle without a GPU.  It is compiled by tests/test_host_replay.py with g++ and is NOT
// part of the library: the product path itself never runs on the CPU.
#include <stdint.h>
#include <string.h>

#include <vector>

#include "../paper_2405_04690_b200/csrc/gb_fast.cuh"
#include "../paper_2405_04690_b200/csrc/gb_fft.cuh"
#include "../paper_2405_04690_b200/csrc/gb_tables.hpp"

using namespace gbk;

namespace {

// one stage for both channels: threads [0, H) own channel A, threads [H, 2H) own channel E
template <int N, int R, int Ns, bool LAST>
void replay_stage(cx* bA, cx* bE, const cx* tw) {
    constexpr int G = Plan<N>::G, H = G / 2;
    std::vector<StageRegs<N, R>> regs(G);
    for (int tid = 0; tid < G; tid++) fft_stage_read<N, R>(tid < H ? bA : bE, tid % H, regs[tid]);
    // (barrier)
    for (int tid = 0; tid < G; tid++) {
        fft_stage_compute<N, R, Ns>(tw, tid % H, regs[tid]);
        cx* buf = tid < H ? bA : bE;
        if (!LAST) {
            fft_stage_store<N, R, Ns>(buf, tid % H, regs[tid]);
        } else {   // the kernels keep these in registers: bin j = ht + H m
            cx h[N / H];
            fft_last_to_bins<N, R>(regs[tid], h);
            for (int m = 0; m < N / H; m++) buf[pad_idx<N>(tid % H + H * m)] = h[m];
        }
    }
    // (barrier)
}
#define REPLAY_X(N_, R_, Ns_) replay_stage<N_, R_, Ns_, false>(bA, bE, tw);
#define REPLAY_L(N_, R_, Ns_) replay_stage<N_, R_, Ns_, true>(bA, bE, tw);

template <int N>
void replay_fft(cx* bA, cx* bE, const cx* tw);
template <> void replay_fft<128>(cx* bA, cx* bE, const cx* tw) { GB_FFT_PLAN_128(REPLAY_X, REPLAY_L) }
template <> void replay_fft<256>(cx* bA, cx* bE, const cx* tw) { GB_FFT_PLAN_256(REPLAY_X, REPLAY_L) }
template <> void replay_fft<512>(cx* bA, cx* bE, const cx* tw) { GB_FFT_PLAN_512(REPLAY_X, REPLAY_L) }
template <> void replay_fft<1024>(cx* bA, cx* bE, const cx* tw) { GB_FFT_PLAN_1024(REPLAY_X, REPLAY_L) }

template <int N>
int replay(const double* params, const OrbitParams& op, int path, double* AE, int64_t* kmin, int* used_fast) {
    constexpr int G = Plan<N>::G;
    const double Tobs = op.Tobs, tau = op.armlength / kCLight;
    std::vector<double> orbit((size_t)kOrbitRows * N);
    build_orbit_table(op, N, orbit.data());
    std::vector<double> twd(2 * kTwiddleN);
    build_twiddles(twd.data());
    const cx* tw = reinterpret_cast<const cx*>(twd.data());
    SrcConst s;
    source_constants(params, Tobs, tau, N, s);
    const bool ok = fast_path_ok(params, Tobs, tau, op.au / kCLight);
    const bool fast = path == 1 || (path == 2 && ok);
    *used_fast = fast ? 1 : 0;
    *kmin = s.kmin;
    std::vector<cx> bufA(padded_len<N>()), bufE(padded_len<N>());
    const double dtN = Tobs / (double)N;
    for (int tid = 0; tid < G; tid++) {
        const double scale = (tid & 1) ? -Tobs / (2.0 * N) : Tobs / (2.0 * N);
        for (int j = 0; j < N / G; j++) {
            const int n = tid + G * j;
            cd As, Es;
            if (fast) {
                OrbitSampleAB o;
                o.Rx = orbit[0 * N + n];
                o.Ry = orbit[1 * N + n];
                for (int d = 0; d < 3; d++) {
                    o.a[d] = orbit[(2 + d) * N + n];
                    o.b[d] = orbit[(5 + d) * N + n];
                }
                slow_sample_fast(s, o, (double)n * dtN, (double)n * (1.0 / N), tau, scale, As, Es);
            } else {
                OrbitSample o;
                o.Rx = orbit[0 * N + n];
                o.Ry = orbit[1 * N + n];
                for (int d = 0; d < 3; d++) {
                    o.a[d] = orbit[(2 + d) * N + n];
                    o.b[d] = orbit[(5 + d) * N + n];
                    o.c[d] = orbit[(8 + d) * N + n];
                }
                slow_sample(s, o, (double)n * dtN, (double)n * (1.0 / N), tau, scale, As, Es);
            }
            bufA[pad_idx<N>(n)] = {As.re, As.im};
            bufE[pad_idx<N>(n)] = {Es.re, Es.im};
        }
    }
    replay_fft<N>(bufA.data(), bufE.data(), tw);
    for (int j = 0; j < N; j++) {
        AE[2 * j] = bufA[pad_idx<N>(j)].re;
        AE[2 * j + 1] = bufA[pad_idx<N>(j)].im;
        AE[2 * (N + j)] = bufE[pad_idx<N>(j)].re;
        AE[2 * (N + j) + 1] = bufE[pad_idx<N>(j)].im;
    }
    return 0;
}

}  // namespace

extern "C" {

// path: 0 = general (slow_sample), 1 = fast (slow_sample_fast) regardless of its limits, 2 = as gb_prep_kernel decides
// AE: [2][N] complex128 interleaved.  Returns 0, or -1 for an unsupported N.
int gb_replay_waveform(const double* params, int N, double Tobs, double armlength, double au, double year,
                       double kappa, double lambda0, int path, double* AE, int64_t* kmin, int* used_fast) {
    const OrbitParams op{Tobs, armlength, au, year, kappa, lambda0};
    switch (N) {
        case 128: return replay<128>(params, op, path, AE, kmin, used_fast);
        case 256: return replay<256>(params, op, path, AE, kmin, used_fast);
        case 512: return replay<512>(params, op, path, AE, kmin, used_fast);
        case 1024: return replay<1024>(params, op, path, AE, kmin, used_fast);
    }
    return -1;
}

// bounded-range sin/cos of the fast path, for the accuracy test: which = 0 (|x|<=0.8), 1 (|x|<=0.27), 2 (reduced)
void gb_replay_sincos(int which, const double* x, int n, double* s, double* c) {
    for (int i = 0; i < n; i++) {
        if (which == 0) sincos_w(x[i], s[i], c[i]);
        else if (which == 1) sincos_n(x[i], s[i], c[i]);
        else sincos_cw(x[i], s[i], c[i]);
    }
}

int gb_replay_fast_ok(const double* params, double Tobs, double armlength, double au) {
    return fast_path_ok(params, Tobs, armlength / kCLight, au / kCLight) ? 1 : 0;
}

}  // extern "C"
