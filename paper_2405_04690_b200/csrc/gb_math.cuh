// gb_math.cuh -- per-source and per-time-sample arithmetic of the GB slow part (product path).
//
// Everything here is written from DESIGN.md "The path" (steps O1-O5), restructured for the FP64 pipe of
// sm_100a; it shares no code with oracle/.  The functions are __host__ __device__ only so that the host
// logic tests can exercise the arithmetic without a GPU; the library itself never runs them on the CPU.
#pragma once
#include <math.h>
#include <stdint.h>

#if defined(__CUDACC__)
#define GB_HD __host__ __device__ __forceinline__
#else
#define GB_HD inline
#endif

namespace gbk {

constexpr double kCLight = 299792458.0;
constexpr double kPi = 3.141592653589793238462643383279502884;
constexpr double kTwoPi = 6.283185307179586476925286766559005768;

struct cd {
    double re, im;
};
GB_HD cd cmul(cd a, cd b) { return {a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re}; }
GB_HD cd cadd(cd a, cd b) { return {a.re + b.re, a.im + b.im}; }
GB_HD cd csub(cd a, cd b) { return {a.re - b.re, a.im - b.im}; }
GB_HD cd cscale(double s, cd a) { return {s * a.re, s * a.im}; }

// product rounded to double before anything is added to it (the carrier bin q must not see an FMA)
GB_HD double mul_rn(double a, double b) {
#if defined(__CUDA_ARCH__)
    return __dmul_rn(a, b);
#else
    volatile double p = a * b;
    return p;
#endif
}

GB_HD void sincos_full(double x, double* s, double* c) {
#if defined(__CUDA_ARCH__)
    sincos(x, s, c);
#else
    *s = sin(x);
    *c = cos(x);
#endif
}

// Per-source constants (step O1 plus the source-only factors of O4).  24 doubles = 192 bytes.
struct SrcConst {
    double k[3];        // propagation direction
    double u[3];        // polarisation basis vector u
    double v[2];        // polarisation basis vector v (v_z = 0)
    cd DP, DC2;         // polarisation constants; DC2 = 2 DC (the factor 2 of d_cross = 2 nu_u nu_v)
    double w0;          // 2 pi f0
    double pifd;        // pi fdot
    double c1;          // (2/3) fdot / f0
    double phi0;
    double twopidelta;  // 2 pi (f0 T - q)
    double hx0;         // pi f0 L / c      (x/2 at t = 0, x = 2 pi f L/c)
    double hxd;         // pi fdot L / c
    int64_t kmin;       // q - N/2
    int32_t fast;       // 1: inside the limits of slow_sample_fast (gb_fast.cuh)
    // row metadata copied in by gb_prep_kernel so that one 192-byte record is all a CTA needs per item
    int32_t move;       // GB_ADD / GB_REMOVE / GB_SWAP
    int32_t walker;     // residual row
    int32_t psd_row;    // PSD row of that walker
    double ch0, sh0;    // cos, sin of hx0 (the fast path rotates them by the tiny angle hxd t instead of a sincos per sample)
};
static_assert(sizeof(SrcConst) == 192, "SrcConst layout");

// Orbit quantities at one time sample (step O2, split about the guiding centre):
// R/c in seconds (z = 0) and the three link unit vectors a = n_12, b = n_23, c = n_31, n_rs = (x_r - x_s)/L.
struct OrbitSample {
    double Rx, Ry;
    double a[3], b[3], c[3];
};

GB_HD void source_constants(const double* p, double Tobs, double tau, int N, SrcConst& s) {
    const double amp = p[0], f0 = p[1], fdot = p[2], phi0 = p[3], ci = p[4], psi = p[5], lam = p[6], sinb = p[7];
    const double cosb = sqrt(1.0 - sinb * sinb);
    double sl, cl, s2p, c2p;
    sincos_full(lam, &sl, &cl);
    sincos_full(2.0 * psi, &s2p, &c2p);
    s.u[0] = sinb * cl;  s.u[1] = sinb * sl;  s.u[2] = -cosb;
    s.v[0] = sl;         s.v[1] = -cl;
    s.k[0] = -cosb * cl; s.k[1] = -cosb * sl; s.k[2] = -sinb;
    const double Ap = amp * (1.0 + ci * ci), Ac = -2.0 * amp * ci;
    s.DP = {Ap * c2p, -Ac * s2p};
    s.DC2 = {-2.0 * Ap * s2p, -2.0 * Ac * c2p};
    const double q = floor(mul_rn(f0, Tobs) + 0.5);
    const double delta = fma(f0, Tobs, -q);
    s.w0 = kTwoPi * f0;
    s.pifd = kPi * fdot;
    s.c1 = (2.0 / 3.0) * (fdot / f0);
    s.phi0 = phi0;
    s.twopidelta = kTwoPi * delta;
    s.hx0 = kPi * f0 * tau;
    s.hxd = kPi * fdot * tau;
    s.kmin = (int64_t)q - N / 2;
    s.fast = 0;
    s.walker = s.psd_row = s.move = 0;
    sincos_full(s.hx0, &s.sh0, &s.ch0);
}

GB_HD double sinc_plain(double th, double sn) { return fabs(th) < 1e-8 ? 1.0 - th * th / 6.0 : sn / th; }

// T_rs = sinc(theta) exp(-i theta)
GB_HD cd transfer(double th) {
    double sn, cs;
    sincos_full(th, &sn, &cs);
    const double sc = sinc_plain(th, sn);
    return {sc * cs, -sc * sn};
}

// Slow envelopes A_s(t_n), E_s(t_n) (steps O3-O5) times `scale`.
//   t      = n T / N,  nfrac = n / N,  tau = L / c
//   scale  = +-T/(2N): the sign (-1)^n moves bin q to the centre of the FFT output (fftshift for free)
GB_HD void slow_sample(const SrcConst& s, const OrbitSample& o, double t, double nfrac, double tau,
                       double scale, cd& As, cd& Es) {
    // link geometry (O3).  The opposite direction of a link flips the sign of nu_u, nu_v, kappa, so
    // d_plus, d_cross and hence D are shared by both directions.
    const double ka = s.k[0] * o.a[0] + s.k[1] * o.a[1] + s.k[2] * o.a[2];
    const double kb = s.k[0] * o.b[0] + s.k[1] * o.b[1] + s.k[2] * o.b[2];
    const double kc = s.k[0] * o.c[0] + s.k[1] * o.c[1] + s.k[2] * o.c[2];
    const double ua = s.u[0] * o.a[0] + s.u[1] * o.a[1] + s.u[2] * o.a[2];
    const double ub = s.u[0] * o.b[0] + s.u[1] * o.b[1] + s.u[2] * o.b[2];
    const double uc = s.u[0] * o.c[0] + s.u[1] * o.c[1] + s.u[2] * o.c[2];
    const double va = s.v[0] * o.a[0] + s.v[1] * o.a[1];
    const double vb = s.v[0] * o.b[0] + s.v[1] * o.b[1];
    const double vc = s.v[0] * o.c[0] + s.v[1] * o.c[1];
    const double dpa = ua * ua - va * va, dca = ua * va;   // the factor 2 of d_cross is in DC2
    const double dpb = ub * ub - vb * vb, dcb = ub * vb;
    const double dpc = uc * uc - vc * vc, dcc = uc * vc;
    const cd Da = {dpa * s.DP.re + dca * s.DC2.re, dpa * s.DP.im + dca * s.DC2.im};   // D_12 = D_21
    const cd Db = {dpb * s.DP.re + dcb * s.DC2.re, dpb * s.DP.im + dcb * s.DC2.im};   // D_23 = D_32
    const cd Dc = {dpc * s.DP.re + dcc * s.DC2.re, dpc * s.DP.im + dcc * s.DC2.im};   // D_31 = D_13

    // k.x_r / c = k.R/c + (tau/3) * (kappa of the two links leaving r), since x_r = R + (L/3)(n_rs + n_rs')
    const double kR = s.k[0] * o.Rx + s.k[1] * o.Ry;
    const double t3 = tau * (1.0 / 3.0);
    const double kx1 = kR + t3 * (ka - kc), kx2 = kR + t3 * (kb - ka), kx3 = kR + t3 * (kc - kb);

    // phases and amplitudes of the three receivers (O4)
    cd G1, G2, G3;
    {
        const double base = s.twopidelta * nfrac + s.phi0;
        const double xi1 = t - kx1, xi2 = t - kx2, xi3 = t - kx3;
        double sn, cs;
        sincos_full(base - s.w0 * kx1 + s.pifd * xi1 * xi1, &sn, &cs);
        const double a1 = 1.0 + s.c1 * xi1;
        G1 = {a1 * cs, a1 * sn};
        sincos_full(base - s.w0 * kx2 + s.pifd * xi2 * xi2, &sn, &cs);
        const double a2 = 1.0 + s.c1 * xi2;
        G2 = {a2 * cs, a2 * sn};
        sincos_full(base - s.w0 * kx3 + s.pifd * xi3 * xi3, &sn, &cs);
        const double a3 = 1.0 + s.c1 * xi3;
        G3 = {a3 * cs, a3 * sn};
    }

    // transfer functions of the six links: theta_rs = x/2 (1 - kappa_rs)
    const double hx = s.hx0 + s.hxd * t;
    const double x = 2.0 * hx;
    const cd T12 = transfer(hx * (1.0 - ka)), T21 = transfer(hx * (1.0 + ka));
    const cd T23 = transfer(hx * (1.0 - kb)), T32 = transfer(hx * (1.0 + kb));
    const cd T31 = transfer(hx * (1.0 - kc)), T13 = transfer(hx * (1.0 + kc));

    // W_rs = T_rs D_pair G_r ;  Y_rs = -(i/2) x W_rs  (the common factor is applied once at the end)
    const cd DG1a = cmul(Da, G1), DG2a = cmul(Da, G2);
    const cd DG2b = cmul(Db, G2), DG3b = cmul(Db, G3);
    const cd DG3c = cmul(Dc, G3), DG1c = cmul(Dc, G1);
    const cd W12 = cmul(T12, DG1a), W21 = cmul(T21, DG2a);
    const cd W23 = cmul(T23, DG2b), W32 = cmul(T32, DG3b);
    const cd W31 = cmul(T31, DG3c), W13 = cmul(T13, DG1c);

    // first-generation Michelson (O5) without the common factor (1 - E1^2):
    //   X' = (W13 - W12) + E1 (W31 - W21), cyclic for Y', Z'
    double sx, cx;
    sincos_full(x, &sx, &cx);
    const cd E1 = {cx, -sx};
    const cd Xp = cadd(csub(W13, W12), cmul(E1, csub(W31, W21)));
    const cd Yp = cadd(csub(W21, W23), cmul(E1, csub(W12, W32)));
    const cd Zp = cadd(csub(W32, W31), cmul(E1, csub(W23, W13)));
    // common factor F = -(i/2) x (1 - E1^2) * scale
    const cd E1sq = cmul(E1, E1);
    const cd om = {1.0 - E1sq.re, -E1sq.im};
    const double hs = 0.5 * x * scale;
    const cd F = {hs * om.im, -hs * om.re};          // -(i) * om * hs
    const cd Ap = csub(Zp, Xp);                                      // sqrt2 A'
    const cd Ep = {Xp.re - 2.0 * Yp.re + Zp.re, Xp.im - 2.0 * Yp.im + Zp.im};   // sqrt6 E'
    As = cscale(0.70710678118654752440, cmul(F, Ap));
    Es = cscale(0.40824829046386301637, cmul(F, Ep));
}

}  // namespace gbk
