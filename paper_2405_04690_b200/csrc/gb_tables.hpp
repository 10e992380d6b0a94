// gb_tables.hpp -- host-side construction of the per-context tables (product path; no oracle code).
//
//  * orbit table for a window length N: SoA [11][N] doubles, rows = Rx/c, Ry/c, a_xyz, b_xyz, c_xyz at
//    t_n = n Tobs / N.  Analytic equal-arm orbits to first order in the eccentricity (O2),
//    written about the guiding centre R = AU (cos alpha, sin alpha, 0) so that the link vectors
//    n_rs = (x_r - x_s)/L are formed from the small offsets r_i = x_i - R without cancellation.
//  * FFT twiddles: tw[k] = exp(-2 pi i k / 1024), k = 0..1023, rounded from long double.
#pragma once
#include <math.h>
#include <vector>

namespace gbk {

constexpr int kOrbitRows = 11;
constexpr int kTwiddleN = 1024;

struct OrbitParams {
    double Tobs, armlength, au, year, kappa, lambda0;
};

inline void build_orbit_table(const OrbitParams& c, int N, double* out /* [11][N] */) {
    const long double PI = 3.141592653589793238462643383279502884L;
    const long double ecc = (long double)c.armlength / (2.0L * sqrtl(3.0L) * (long double)c.au);
    const long double clight = 299792458.0L;
    for (int n = 0; n < N; n++) {
        const long double t = (long double)n * (long double)c.Tobs / (long double)N;
        const long double al = 2.0L * PI * t / (long double)c.year + (long double)c.kappa;
        const long double sa = sinl(al), ca = cosl(al);
        long double r[3][3];
        for (int i = 0; i < 3; i++) {
            const long double be = 2.0L * PI * i / 3.0L + (long double)c.lambda0;
            const long double sb = sinl(be), cb = cosl(be);
            r[i][0] = c.au * ecc * (sa * ca * sb - (1.0L + sa * sa) * cb);
            r[i][1] = c.au * ecc * (sa * ca * cb - (1.0L + ca * ca) * sb);
            r[i][2] = -sqrtl(3.0L) * c.au * ecc * cosl(al - be);
        }
        out[0 * N + n] = (double)(c.au * ca / clight);
        out[1 * N + n] = (double)(c.au * sa / clight);
        const int pr[3][2] = {{0, 1}, {1, 2}, {2, 0}};   // a = n_12, b = n_23, c = n_31
        for (int l = 0; l < 3; l++)
            for (int d = 0; d < 3; d++)
                out[(2 + 3 * l + d) * N + n] = (double)((r[pr[l][0]][d] - r[pr[l][1]][d]) / (long double)c.armlength);
    }
}

inline void build_twiddles(double* out /* [1024][2] */) {
    const long double PI = 3.141592653589793238462643383279502884L;
    for (int k = 0; k < kTwiddleN; k++) {
        const long double ang = 2.0L * PI * (long double)k / (long double)kTwiddleN;
        out[2 * k] = (double)cosl(ang);
        out[2 * k + 1] = (double)(-sinl(ang));
    }
}

}  // namespace gbk
