// gb_fast.cuh -- the slow part (steps O2-O5 of DESIGN.md) restructured for the FP64 pipe of sm_100a.
//
// Same definition as slow_sample() in gb_math.cuh, evaluated with 3 polynomial sin/cos pairs, one small-angle
// rotation of a per-source constant, no division by an angle and one shared reciprocal per time sample instead of
// 10 library sincos + 6 divisions:
//
//   * a + b + c = 0 for the three link vectors, so kappa_c, nu_u,c, nu_v,c follow from the a and b links;
//   * with psi_l = x kappa_l / 6 (x = 2 pi (f0 + fdot t) L/c) every angle of the response is an integer
//     combination of x/2, psi_a, psi_b:   theta_rs = x/2 -+ 3 psi_l,   and the receiver phase offsets are
//     -(x/3)(kappa_l - kappa_l') = -2 (psi_l - psi_l') up to eps_r = pi fdot d_r (2 k.R/c + d_r) (< 1e-8 rad,
//     first order).  Double/triple-angle formulas (relative accuracy kept for small sines) and complex
//     products give all phasors from exp(i x/2), sincos(psi_a), sincos(psi_b) -- small, bounded arguments
//     that need no range reduction (gb_sincos_poly.h); exp(i x/2) itself is the per-source constant exp(i x0/2)
//     rotated by the tiny angle pi fdot t L/c (series);
//   * (x/2) sinc(theta_rs) = sin(theta_rs) / (1 - kappa_rs): the six denominators share one reciprocal of
//     (1-kappa_a^2)(1-kappa_b^2)(1-kappa_c^2); a link within ~1e-2 rad of the source direction takes the
//     series of sinc instead (rare branch);
//   * the phase common to all links, Phi_R = 2 pi delta n/N + phi0 - 2 pi f0 k.R/c + pi fdot (t - k.R/c)^2,
//     is factored out of X, Y, Z and applied once: one Cody-Waite reduced sincos;
//   * 1 - E1^2 = 2 i sin(x) E1.
//
// Valid when fast_path_ok() holds (|x|/2 <= 0.8 i.e. f0 <~ 30.5 mHz, |fdot| small enough for eps_r < 1e-8,
// |Phi_R| < 3000); gb_prep_kernel routes every other row to the general kernels built on slow_sample().
#pragma once
#include "gb_math.cuh"
#include "gb_sincos_poly.h"

namespace gbk {

// Numeric constants of the fast path.  On the device they sit in __constant__ memory so that every use is a
// c[bank][offset] operand of the DFMA / DMUL itself: a 64-bit literal would cost two extra issue slots (a pair
// of 32-bit moves) per use, and the issue slot is the second bound of this kernel after the FP64 pipe.
struct FastConsts {
    double wS[6], wC[6];   // |x| <= 0.8
    double nS[5], nC[4];   // |x| <= 0.27
    double two_over_pi, pio2_hi, pio2_lo;
    double third, rsqrt2, rsqrt3, r120, msixth, r24;
};
#define GB_FAST_CONSTS_INIT                                                                                   \
    {GB_POLY_W_SIN, GB_POLY_W_COS, GB_POLY_N_SIN, GB_POLY_N_COS, GB_TWO_OVER_PI, GB_PIO2_HI, GB_PIO2_LO,      \
     1.0 / 3.0, 0.70710678118654752440, 0.57735026918962576451, 1.0 / 120.0, -1.0 / 6.0, 1.0 / 24.0}
#if defined(__CUDACC__)
__constant__ FastConsts d_fast_consts = GB_FAST_CONSTS_INIT;
#endif
static const FastConsts h_fast_consts = GB_FAST_CONSTS_INIT;
#if defined(__CUDA_ARCH__)
#define GB_K(field) (d_fast_consts.field)
#else
#define GB_K(field) (h_fast_consts.field)
#endif

// sin, cos for |x| <= 0.8 (no range reduction)
GB_HD void sincos_w(double x, double& s, double& c) {
    const double z = x * x;
    double ps = fma(GB_K(wS[5]), z, GB_K(wS[4]));
    double pc = fma(GB_K(wC[5]), z, GB_K(wC[4]));
    ps = fma(ps, z, GB_K(wS[3]));
    pc = fma(pc, z, GB_K(wC[3]));
    ps = fma(ps, z, GB_K(wS[2]));
    pc = fma(pc, z, GB_K(wC[2]));
    ps = fma(ps, z, GB_K(wS[1]));
    pc = fma(pc, z, GB_K(wC[1]));
    ps = fma(ps, z, GB_K(wS[0]));
    pc = fma(pc, z, GB_K(wC[0]));
    s = fma(x * z, ps, x);
    c = fma(z, fma(z, pc, -0.5), 1.0);
}

// sin, cos for |x| <= 0.27
GB_HD void sincos_n(double x, double& s, double& c) {
    const double z = x * x;
    double ps = fma(GB_K(nS[4]), z, GB_K(nS[3]));
    double pc = fma(GB_K(nC[3]), z, GB_K(nC[2]));
    ps = fma(ps, z, GB_K(nS[2]));
    pc = fma(pc, z, GB_K(nC[1]));
    ps = fma(ps, z, GB_K(nS[1]));
    pc = fma(pc, z, GB_K(nC[0]));
    ps = fma(ps, z, GB_K(nS[0]));
    s = fma(x * z, ps, x);
    c = fma(z, fma(z, pc, -0.5), 1.0);
}

GB_HD int lo32_of(double v) {
#if defined(__CUDA_ARCH__)
    return __double2loint(v);
#else
    union { double d; int64_t i; } u;
    u.d = v;
    return (int)(u.i & 0xffffffff);
#endif
}

// sin, cos for |x| < 3000: two-constant Cody-Waite reduction by pi/2, then sincos_w and the quadrant
GB_HD void sincos_cw(double x, double& s, double& c) {
    constexpr double kMagic = 6755399441055744.0;   // 1.5 * 2^52: the low word of x*2/pi + magic is rint()
    const double kd = fma(x, GB_K(two_over_pi), kMagic);
    const int q = lo32_of(kd);
    const double kf = kd - kMagic;
    double r = fma(-kf, GB_K(pio2_hi), x);
    r = fma(-kf, GB_K(pio2_lo), r);
    double sr, cr;
    sincos_w(r, sr, cr);
    double a = (q & 1) ? cr : sr;
    double b = (q & 1) ? sr : cr;
    s = (q & 2) ? -a : a;
    c = ((q + 1) & 2) ? -b : b;
}

GB_HD double rcp_fast(double p) {   // 1/p for normal p > 0 to 1 ulp (measured on B200 over [1e-4, 1]: 2.2e-16)
#if defined(__CUDA_ARCH__)
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(p));   // relative error <= 1e-6
    const double e = fma(-p, y, 1.0);
    return fma(y, fma(e, e, e), y);                         // third-order step: e^3 ~ 1e-18
#else
    return 1.0 / p;
#endif
}

// limits of the fast path (see the header comment); Rmax = AU/c
GB_HD bool fast_path_ok(const double* p, double Tobs, double tau, double Rmax) {
    const double f0 = p[1], fdot = p[2], phi0 = p[3];
    const double hxmax = kPi * tau * (fabs(f0) + fabs(fdot) * Tobs);
    const double dmax = 2.0 * tau / 3.0;
    const double eps = kPi * fabs(fdot) * dmax * (2.0 * Rmax + dmax);
    const double tt = Tobs + Rmax + tau;
    const double ph = fabs(phi0) + kPi + kTwoPi * fabs(f0) * Rmax + kPi * fabs(fdot) * tt * tt;
    return f0 > 0.0 && hxmax <= 0.8 && eps < 1e-8 && ph < 3000.0;   // NaN anywhere -> false
}

// Orbit quantities the fast path reads: R/c and the link vectors a = n_12, b = n_23 (c = -a - b).
struct OrbitSampleAB {
    double Rx, Ry;
    double a[3], b[3];
};

// sin(theta)/(1 -+ kappa) for theta = hx (1 -+ kappa) when 1 -+ kappa = d is tiny: hx sinc(theta)
GB_HD double sinc_guarded(double hx, double sn, double d) {
    if (fabs(d) >= 1e-4) return sn / d;
    const double th = hx * d, z = th * th;
    return hx * fma(z, fma(z, GB_K(r120), GB_K(msixth)), 1.0);
}

// Slow envelopes A_s(t_n), E_s(t_n) times `scale`; arguments as slow_sample().
GB_HD void slow_sample_fast(const SrcConst& s, const OrbitSampleAB& o, double t, double nfrac, double tau,
                            double scale, cd& As, cd& Es) {
    // ---- link geometry (O3)
    const double ka = s.k[0] * o.a[0] + s.k[1] * o.a[1] + s.k[2] * o.a[2];
    const double kb = s.k[0] * o.b[0] + s.k[1] * o.b[1] + s.k[2] * o.b[2];
    const double kc = -(ka + kb);
    const double ua = s.u[0] * o.a[0] + s.u[1] * o.a[1] + s.u[2] * o.a[2];
    const double ub = s.u[0] * o.b[0] + s.u[1] * o.b[1] + s.u[2] * o.b[2];
    const double uc = -(ua + ub);
    const double va = s.v[0] * o.a[0] + s.v[1] * o.a[1];
    const double vb = s.v[0] * o.b[0] + s.v[1] * o.b[1];
    const double vc = -(va + vb);
    const double dpa = ua * ua - va * va, dca = ua * va;   // DC2 = 2 DC carries the factor 2 of d_cross
    const double dpb = ub * ub - vb * vb, dcb = ub * vb;
    const double dpc = uc * uc - vc * vc, dcc = uc * vc;
    const cd Da = {dpa * s.DP.re + dca * s.DC2.re, dpa * s.DP.im + dca * s.DC2.im};
    const cd Db = {dpb * s.DP.re + dcb * s.DC2.re, dpb * s.DP.im + dcb * s.DC2.im};
    const cd Dc = {dpc * s.DP.re + dcc * s.DC2.re, dpc * s.DP.im + dcc * s.DC2.im};

    // ---- angles: hx = x/2, psi_l = hx kappa_l / 3
    const double kR = s.k[0] * o.Rx + s.k[1] * o.Ry;
    const double xiR = t - kR;
    const double hx = fma(s.hxd, t, s.hx0);
    const double hx3 = hx * GB_K(third);
    double sh, ch, sa, ca, sb, cb;
    {   // exp(i hx) = exp(i hx0) exp(i eps), eps = hxd t: |eps| < 5e-4 inside the fast limits, series to eps^4 / eps^3
        const double eps = s.hxd * t, e2 = eps * eps;
        const double ce = fma(e2, fma(e2, GB_K(r24), -0.5), 1.0);
        const double se = eps * fma(e2, GB_K(msixth), 1.0);
        sh = fma(s.sh0, ce, s.ch0 * se);
        ch = fma(s.ch0, ce, -(s.sh0 * se));
    }
    sincos_n(hx3 * ka, sa, ca);
    sincos_n(hx3 * kb, sb, cb);
    // double and triple angles of psi_a, psi_b; psi_c = -(psi_a + psi_b) by products
    const double saa = sa * sa, sbb = sb * sb;
    const cd Pa2 = {fma(-2.0, saa, 1.0), (sa + sa) * ca};
    const cd Pb2 = {fma(-2.0, sbb, 1.0), (sb + sb) * cb};
    const cd Pa3 = {ca * fma(-4.0, saa, 1.0), sa * fma(-4.0, saa, 3.0)};
    const cd Pb3 = {cb * fma(-4.0, sbb, 1.0), sb * fma(-4.0, sbb, 3.0)};
    const cd Pc2 = {Pa2.re * Pb2.re - Pa2.im * Pb2.im, -(Pa2.re * Pb2.im + Pa2.im * Pb2.re)};
    const cd Pc3 = {Pa3.re * Pb3.re - Pa3.im * Pb3.im, -(Pa3.re * Pb3.im + Pa3.im * Pb3.re)};

    // ---- receiver factors g_r = a_r exp(i (phase_r - Phi_R)) = Q_r (a_r, a_r eps_r)   (O4)
    //      Q_1 = conj(Pa2) Pc2, Q_2 = conj(Pb2) Pa2, Q_3 = conj(Pc2) Pb2
    const double t3 = tau * GB_K(third);
    const double d1 = t3 * (ka - kc), d2 = t3 * (kb - ka), d3 = t3 * (kc - kb);
    const double aR = fma(s.c1, xiR, 1.0);
    const double a1 = fma(-s.c1, d1, aR), a2 = fma(-s.c1, d2, aR), a3 = fma(-s.c1, d3, aR);
    const double kR2 = kR + kR;
    const double e1 = (s.pifd * d1) * (kR2 + d1);   // eps_r (first order: |eps_r| < 1e-8)
    const double e2 = (s.pifd * d2) * (kR2 + d2);
    const double e3 = (s.pifd * d3) * (kR2 + d3);
    const cd Q1 = {Pa2.re * Pc2.re + Pa2.im * Pc2.im, Pa2.re * Pc2.im - Pa2.im * Pc2.re};
    const cd Q2 = {Pb2.re * Pa2.re + Pb2.im * Pa2.im, Pb2.re * Pa2.im - Pb2.im * Pa2.re};
    const cd Q3 = {Pc2.re * Pb2.re + Pc2.im * Pb2.im, Pc2.re * Pb2.im - Pc2.im * Pb2.re};
    const cd g1 = {a1 * fma(-Q1.im, e1, Q1.re), a1 * fma(Q1.re, e1, Q1.im)};   // a_r Q_r (1 + i eps_r)
    const cd g2 = {a2 * fma(-Q2.im, e2, Q2.re), a2 * fma(Q2.re, e2, Q2.im)};
    const cd g3 = {a3 * fma(-Q3.im, e3, Q3.re), a3 * fma(Q3.re, e3, Q3.im)};

    // ---- transfer: theta_12 = hx - 3 psi_a, theta_21 = hx + 3 psi_a, ...;  T'_rs = sin(th)/(1 - kappa_rs) exp(-i th)
    const double ma = fma(-ka, ka, 1.0), mb = fma(-kb, kb, 1.0), mc = fma(-kc, kc, 1.0);
    const double mab = ma * mb, pp = mab * mc;
    const double inv = rcp_fast(pp);
    const double ra = inv * (mb * mc), rb = inv * (ma * mc), rc = inv * mab;   // 1 / (1 - kappa_l^2)
    // cos / sin of theta for both directions of each link
    const double c12 = fma(sh, Pa3.im, ch * Pa3.re), s12 = fma(sh, Pa3.re, -(ch * Pa3.im));
    const double c21 = fma(-sh, Pa3.im, ch * Pa3.re), s21 = fma(sh, Pa3.re, ch * Pa3.im);
    const double c23 = fma(sh, Pb3.im, ch * Pb3.re), s23 = fma(sh, Pb3.re, -(ch * Pb3.im));
    const double c32 = fma(-sh, Pb3.im, ch * Pb3.re), s32 = fma(sh, Pb3.re, ch * Pb3.im);
    const double c31 = fma(sh, Pc3.im, ch * Pc3.re), s31 = fma(sh, Pc3.re, -(ch * Pc3.im));
    const double c13 = fma(-sh, Pc3.im, ch * Pc3.re), s13 = fma(sh, Pc3.re, ch * Pc3.im);
    double q12 = s12 * ((1.0 + ka) * ra), q21 = s21 * ((1.0 - ka) * ra);
    double q23 = s23 * ((1.0 + kb) * rb), q32 = s32 * ((1.0 - kb) * rb);
    double q31 = s31 * ((1.0 + kc) * rc), q13 = s13 * ((1.0 - kc) * rc);
    if (!(pp >= 1e-4)) {   // a link nearly along the source direction (or NaN input): series for that link
        q12 = sinc_guarded(hx, s12, 1.0 - ka);   // (the shared reciprocal may have overflowed: plain divisions)
        q21 = sinc_guarded(hx, s21, 1.0 + ka);
        q23 = sinc_guarded(hx, s23, 1.0 - kb);
        q32 = sinc_guarded(hx, s32, 1.0 + kb);
        q31 = sinc_guarded(hx, s31, 1.0 - kc);
        q13 = sinc_guarded(hx, s13, 1.0 + kc);
    }

    // ---- W'_rs = T'_rs D_pair g_r  (= hx W_rs of slow_sample)
    const cd DG1a = cmul(Da, g1), DG2a = cmul(Da, g2);
    const cd DG2b = cmul(Db, g2), DG3b = cmul(Db, g3);
    const cd DG3c = cmul(Dc, g3), DG1c = cmul(Dc, g1);
    const cd W12 = cmul({q12 * c12, -(q12 * s12)}, DG1a), W21 = cmul({q21 * c21, -(q21 * s21)}, DG2a);
    const cd W23 = cmul({q23 * c23, -(q23 * s23)}, DG2b), W32 = cmul({q32 * c32, -(q32 * s32)}, DG3b);
    const cd W31 = cmul({q31 * c31, -(q31 * s31)}, DG3c), W13 = cmul({q13 * c13, -(q13 * s13)}, DG1c);

    // ---- first-generation Michelson (O5): X' = (W13 - W12) + E1 (W31 - W21), cyclic
    const double sx = (sh + sh) * ch, cx = fma(-2.0 * sh, sh, 1.0);
    const cd E1 = {cx, -sx};
    const cd Xp = cadd(csub(W13, W12), cmul(E1, csub(W31, W21)));
    const cd Yp = cadd(csub(W21, W23), cmul(E1, csub(W12, W32)));
    const cd Zp = cadd(csub(W32, W31), cmul(E1, csub(W23, W13)));

    // ---- common factor: -(i) scale (1 - E1^2) exp(i Phi_R) = 2 scale sin(x) E1 exp(i Phi_R)
    double sR, cR;
    sincos_cw(fma(s.twopidelta, nfrac, s.phi0) - s.w0 * kR + s.pifd * xiR * xiR, sR, cR);
    const double f2 = (2.0 * GB_K(rsqrt2)) * scale * sx;                           // 1/sqrt2 of A folded in
    const cd F = cmul({f2 * cx, -(f2 * sx)}, {cR, sR});
    const cd Ap = csub(Zp, Xp);                                                    // sqrt2 A'
    const cd Ep = {Xp.re - 2.0 * Yp.re + Zp.re, Xp.im - 2.0 * Yp.im + Zp.im};      // sqrt6 E'
    As = cmul(F, Ap);
    Es = cscale(GB_K(rsqrt3), cmul(F, Ep));
}

}  // namespace gbk
