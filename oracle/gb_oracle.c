/*
 * gb_oracle.c -- CPU ORACLE for the Galactic-binary (GB) waveform + delta-log-likelihood hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call it.  The CUDA product
 * path (paper_2405_04690_b200/) shares no code, header, table or constant generator with this file
 * and never calls it.
 *
 * What it computes (plain, slow, fp64, in the paper's order and notation):
 *   the GB frequency-domain TDI A/E waveform by the fast/slow decomposition (sec. II.A,
 *   PAPER.md:696-704 App. F), TDI generation 1.5 with equal constant arms, A/E channels
 *   (Eq. 6), the noise-weighted inner product (Eq. 2), the add / swap
 *   delta log-likelihoods (Eq. 4, 5) and the residual refresh of Algorithm 1
 *   (PAPER.md:599-613).  The paper does not print the waveform equations; the reading
 *   followed here is SURVEY.md sec. 8(c) steps O1..O9 (restated in DESIGN.md "Readings").
 *
 * Style rules: one function per step O1..O9, C99 complex arithmetic so each line reads like the
 * formula, no blocking, no fusion, no reordering, no tables shared between sources.  Compile with
 * -ffp-contract=off so that q = floor(fl(f0*T)+0.5) is rounded as written (reading S4).
 * The only parallelism is an OpenMP "parallel for" over independent proposals / walkers, which does
 * not change any result bit.
 *
 * Pins (tests/test_oracle_pins.py, all -m "not gpu"): frozen-geometry time-domain TDI + DFT (P1),
 * decimation identity (P1'), full-rate dt*rfft (P2), moving geometry (P3), Parseval (P4),
 * monochromatic closed form (P5), delta-lnL invariants (P6), tiny-T brute force (P8); per-channel noise rows
 * (S_E = 4 S_A against the numpy sums); Philox4x32-10 known-answer vectors, the stretch density's closed-form CDF,
 * friends against a numpy argsort, and the z^(D-1) factor by sampling an 8-dimensional Gaussian with the generated
 * proposals (the proposal step of Algorithm 1).
 * "parity unpinned": physical fidelity to the LDC Sangria generator / GBGPU (neither is in this
 * container); the oracle, not those codes, defines the result.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define GBO_C_LIGHT 299792458.0
#define GBO_PI 3.14159265358979323846264338327950288

typedef struct {
    double Tobs;      /* observation time T [s]                    (31457280)            */
    double dt;        /* sampling cadence of the data [s]          (5); not used by O1-O6 */
    double armlength; /* L [m]                                     (2.5e9)               */
    double au;        /* AU [m]                                    (1.495978707e11)      */
    double year;      /* sidereal year [s]                         (31558149.763545603)  */
    double kappa;     /* initial orbital phase of the guiding centre                     */
    double lambda0;   /* initial orientation of the constellation                        */
} gbo_config;

typedef struct {          /* host-resident data view; mirrors the product's gb_data but is its own type */
    double *resid;        /* [n_walkers][2][n_f] complex128 interleaved (r = d - H)                     */
    const double *psd;    /* [n_psd][2][n_f] f64; S_n, or 1/S_n if psd_is_inverse                       */
    const int32_t *walker_psd; /* [n_walkers] -> psd row; NULL = identity (or row 0 if n_psd == 1)      */
    int64_t k_lo, n_f;    /* residual element i <-> global bin k_lo + i                                  */
    int32_t n_walkers, n_psd, psd_is_inverse;
} gbo_data;

enum { GBO_ADD = 0, GBO_REMOVE = 1, GBO_SWAP = 2 };
enum { GBO_OK = 0, GBO_ERR_INVALID = -1 };

void gbo_default_config(gbo_config *c) {
    c->Tobs = 31457280.0;
    c->dt = 5.0;
    c->armlength = 2.5e9;
    c->au = 1.495978707e11;
    c->year = 31558149.763545603;
    c->kappa = 0.0;
    c->lambda0 = 0.0;
}

/* params row = [amp, f0, fdot, phi0, cos_iota, psi, lambda, sin_beta]  (reading S3) */
enum { P_AMP = 0, P_F0, P_FDOT, P_PHI0, P_COSI, P_PSI, P_LAM, P_SINB };

typedef struct {
    double u[3], v[3], k[3]; /* polarisation basis and propagation direction */
    double complex DP, DC;   /* polarisation constants                        */
    int64_t q;               /* carrier bin                                   */
    double delta;            /* f0*T - q, cycles                              */
} gbo_source;

/* ---- O1  source constants ---------------------------------------------------- */
static void o1_source_constants(const gbo_config *c, const double *p, gbo_source *s) {
    double sinb = p[P_SINB];
    double cosb = sqrt(1.0 - sinb * sinb);     /* cos(beta) >= 0                                */
    /* theta_c = pi/2 - beta  =>  cos(theta_c) = sin(beta), sin(theta_c) = cos(beta); phi = lambda */
    double costh = sinb, sinth = cosb;
    double cosph = cos(p[P_LAM]), sinph = sin(p[P_LAM]);
    s->u[0] = costh * cosph;  s->u[1] = costh * sinph;  s->u[2] = -sinth;
    s->v[0] = sinph;          s->v[1] = -cosph;         s->v[2] = 0.0;
    s->k[0] = -sinth * cosph; s->k[1] = -sinth * sinph; s->k[2] = -costh;
    double amp = p[P_AMP], ci = p[P_COSI];
    double Ap = amp * (1.0 + ci * ci);         /* A_plus  */
    double Ac = -2.0 * amp * ci;               /* A_cross */
    double c2p = cos(2.0 * p[P_PSI]), s2p = sin(2.0 * p[P_PSI]);
    s->DP = Ap * c2p - I * (Ac * s2p);
    s->DC = -Ap * s2p - I * (Ac * c2p);
    double prod = p[P_F0] * c->Tobs;           /* rounded product (no FMA contraction)          */
    s->q = (int64_t)floor(prod + 0.5);
    s->delta = fma(p[P_F0], c->Tobs, -(double)s->q);
}

/* ---- O2  analytic equal-arm orbits, first order in eccentricity -------------- */
static void o2_orbits(const gbo_config *c, double t, double x[3][3]) {
    double fm = 1.0 / c->year;
    double ecc = c->armlength / (2.0 * sqrt(3.0) * c->au);
    double alpha = 2.0 * GBO_PI * fm * t + c->kappa;
    double sa = sin(alpha), ca = cos(alpha);
    for (int i = 0; i < 3; i++) {              /* spacecraft i+1 */
        double beta = 2.0 * GBO_PI * i / 3.0 + c->lambda0;
        double sb = sin(beta), cb = cos(beta);
        x[i][0] = c->au * ca + c->au * ecc * (sa * ca * sb - (1.0 + sa * sa) * cb);
        x[i][1] = c->au * sa + c->au * ecc * (sa * ca * cb - (1.0 + ca * ca) * sb);
        x[i][2] = -sqrt(3.0) * c->au * ecc * cos(alpha - beta);
    }
}

static double dot3(const double a[3], const double b[3]) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }

static double sinc(double th) {
    if (fabs(th) < 1e-8) return 1.0 - th * th / 6.0;
    return sin(th) / th;
}

/* ---- O3 + O4 + O5  slow envelope of A and E at time sample n of N ---- */
static void slow_envelope(const gbo_config *c, const double *p, const gbo_source *src, int N, int n,
                          double *As_out, double *Es_out) {
    const gbo_source s = *src;
    double T = c->Tobs, L = c->armlength;
    double f0 = p[P_F0], fdot = p[P_FDOT], phi0 = p[P_PHI0];
    double t = (double)n * T / (double)N;
    double x[3][3];
    o2_orbits(c, t, x);

    double xarg = 2.0 * GBO_PI * (f0 + fdot * t) * L / GBO_C_LIGHT;  /* x(t_n), common to all links */
    double complex Y[3][3];                                            /* Y[r][s], receiver r, sender s */
    for (int r = 0; r < 3; r++) {
        double kx = dot3(s.k, x[r]) / GBO_C_LIGHT;                     /* k.x_r / c            */
        double xi = t - kx;                                            /* xi_r                 */
        double a_r = 1.0 + (2.0 / 3.0) * (fdot / f0) * xi;
        double phi = 2.0 * GBO_PI * (s.delta * ((double)n / (double)N) - f0 * kx)
                   + GBO_PI * fdot * xi * xi + phi0;                   /* Phi(xi_r) - 2 pi q t_n / T */
        for (int sd = 0; sd < 3; sd++) {
            if (sd == r) { Y[r][sd] = 0.0; continue; }
            double nrs[3];                                             /* O3 link vector       */
            for (int d = 0; d < 3; d++) nrs[d] = (x[r][d] - x[sd][d]) / L;
            double nu_u = dot3(s.u, nrs), nu_v = dot3(s.v, nrs), kap = dot3(s.k, nrs);
            double dplus = nu_u * nu_u - nu_v * nu_v;
            double dcross = 2.0 * nu_u * nu_v;
            double complex D = dplus * s.DP + dcross * s.DC;
            double th = 0.5 * xarg * (1.0 - kap);
            Y[r][sd] = -(0.5 * I) * xarg * sinc(th) * cexp(-I * th) * D * a_r * cexp(I * phi);
        }
    }
    /* O5  first-generation Michelson with delay phasor E1 = exp(-i x); indices receiver,sender */
    double complex E1 = cexp(-I * xarg);
    double complex XYZ[3];
    for (int a = 0; a < 3; a++) {              /* a = 0: X (1,2,3), 1: Y (2,3,1), 2: Z (3,1,2) */
        int i1 = a, i2 = (a + 1) % 3, i3 = (a + 2) % 3;
        XYZ[a] = (1.0 - E1 * E1) * ((Y[i1][i3] - Y[i1][i2]) + E1 * (Y[i3][i1] - Y[i2][i1]));
    }
    double complex As = (XYZ[2] - XYZ[0]) / sqrt(2.0);                 /* Eq. 6a */
    double complex Es = (XYZ[0] - 2.0 * XYZ[1] + XYZ[2]) / sqrt(6.0);  /* Eq. 6b */
    As_out[0] = creal(As); As_out[1] = cimag(As);
    Es_out[0] = creal(Es); Es_out[1] = cimag(Es);
}

/* public form: O1 then O3-O5 for one sample (exposed for pins P4, P5) */
void gbo_slow_envelope(const gbo_config *c, const double *p, int N, int n, double *As_out, double *Es_out) {
    gbo_source s;
    o1_source_constants(c, p, &s);
    slow_envelope(c, p, &s, N, n, As_out, Es_out);
}

/* ---- plain O(N^2) DFT, numpy-forward sign:  F[j] = sum_n x[n] exp(-2 pi i j n / N) ------------- */
void gbo_dft(const double *x, int N, double *F) {
    for (int j = 0; j < N; j++) {
        double complex acc = 0.0;
        for (int n = 0; n < N; n++) {
            int m = (int)(((int64_t)j * n) % N);                       /* exact phase reduction */
            double ang = -2.0 * GBO_PI * (double)m / (double)N;
            acc += (x[2 * n] + I * x[2 * n + 1]) * (cos(ang) + I * sin(ang));
        }
        F[2 * j] = creal(acc); F[2 * j + 1] = cimag(acc);
    }
}

/* ---- textbook iterative radix-2 decimation-in-time FFT, same sign; N a power of two ------------ */
int gbo_fft(const double *x, int N, double *F) {
    if (N < 1 || (N & (N - 1))) return GBO_ERR_INVALID;
    int bits = 0; while ((1 << bits) < N) bits++;
    double complex *a = (double complex *)malloc(sizeof(double complex) * (size_t)N);
    for (int n = 0; n < N; n++) {
        int rev = 0;
        for (int b = 0; b < bits; b++) if (n & (1 << b)) rev |= 1 << (bits - 1 - b);
        a[rev] = x[2 * n] + I * x[2 * n + 1];
    }
    for (int len = 2; len <= N; len <<= 1) {
        for (int start = 0; start < N; start += len) {
            for (int m = 0; m < len / 2; m++) {
                double ang = -2.0 * GBO_PI * (double)m / (double)len;
                double complex w = cos(ang) + I * sin(ang);
                double complex e = a[start + m], o = w * a[start + m + len / 2];
                a[start + m] = e + o;
                a[start + m + len / 2] = e - o;
            }
        }
    }
    for (int j = 0; j < N; j++) { F[2 * j] = creal(a[j]); F[2 * j + 1] = cimag(a[j]); }
    free(a);
    return GBO_OK;
}

static int valid_N(int N) { return N >= 2 && N <= (1 << 20) && !(N & (N - 1)); }

/* ---- O6  FFT of the slow part and mapping to bins ------------------------------
 * A[kmin + j] = (T / (2N)) * F[j - N/2],  j = 0..N-1,  kmin = q - N/2,  F indexed modulo N.
 * use_dft != 0 uses the O(N^2) definition instead of the radix-2 FFT (for pins).                  */
int gbo_waveform_ex(const gbo_config *c, const double *p, int N, int use_dft,
                    double *A, double *E, int64_t *kmin) {
    if (!valid_N(N)) return GBO_ERR_INVALID;
    gbo_source s;
    o1_source_constants(c, p, &s);
    double *as = (double *)malloc(sizeof(double) * 2 * (size_t)N * 4);
    double *es = as + 2 * (size_t)N, *Fa = es + 2 * (size_t)N, *Fe = Fa + 2 * (size_t)N;
    for (int n = 0; n < N; n++) slow_envelope(c, p, &s, N, n, as + 2 * n, es + 2 * n);
    if (use_dft) { gbo_dft(as, N, Fa); gbo_dft(es, N, Fe); }
    else         { gbo_fft(as, N, Fa); gbo_fft(es, N, Fe); }
    double scale = c->Tobs / (2.0 * (double)N);
    for (int j = 0; j < N; j++) {
        int jj = (j - N / 2 + N) % N;          /* F[j - N/2] with negative indices wrapped */
        A[2 * j] = scale * Fa[2 * jj]; A[2 * j + 1] = scale * Fa[2 * jj + 1];
        E[2 * j] = scale * Fe[2 * jj]; E[2 * j + 1] = scale * Fe[2 * jj + 1];
    }
    *kmin = s.q - N / 2;
    free(as);
    return GBO_OK;
}

int gbo_waveform(const gbo_config *c, const double *p, int N, double *A, double *E, int64_t *kmin) {
    return gbo_waveform_ex(c, p, N, 0, A, E, kmin);
}

/* batched form of the product's gb_waveform: AE_out [B][2][Nmax] complex128, kmin_out [B] */
int gbo_waveform_batch(const gbo_config *c, const double *params, int64_t B, int N, const int32_t *n_bins,
                       int Nmax, double *AE_out, int64_t *kmin_out, int nthreads) {
    int bad = 0;
#pragma omp parallel for schedule(dynamic, 16) num_threads(nthreads > 0 ? nthreads : 1)
    for (int64_t b = 0; b < B; b++) {
        int Nb = n_bins ? n_bins[b] : N;
        if (!valid_N(Nb) || Nb > Nmax) { bad = 1; continue; }
        double *A = (double *)malloc(sizeof(double) * 4 * (size_t)Nb), *E = A + 2 * (size_t)Nb;
        gbo_waveform(c, params + 8 * b, Nb, A, E, &kmin_out[b]);
        double *outA = AE_out + (size_t)b * 2 * 2 * (size_t)Nmax, *outE = outA + 2 * (size_t)Nmax;
        memcpy(outA, A, sizeof(double) * 2 * (size_t)Nb);
        memcpy(outE, E, sizeof(double) * 2 * (size_t)Nb);
        free(A);
    }
    return bad ? GBO_ERR_INVALID : GBO_OK;
}

/* ---- O7  noise-weighted inner product on aligned windows (Eq. 2) --------------------
 * <b|c> = (4/T) sum_ch sum_k Re[conj(b_ch[k]) c_ch[k]] / S_ch[k] over global bins k that lie in both
 * windows and in the stored band [k_lo, k_lo + n_f)  (reading S13).
 * b: window starting at global bin kb with nb bins, channel arrays bA,bE (interleaved complex);
 * c likewise.  S given by psd row pointers (S or 1/S).                                              */
static double o7_inner(const gbo_config *cfg, const gbo_data *d, int psd_row,
                       const double *bA, const double *bE, int64_t kb, int nb,
                       const double *cA, const double *cE, int64_t kc, int nc) {
    int64_t lo = kb > kc ? kb : kc;
    int64_t hi = (kb + nb) < (kc + nc) ? (kb + nb) : (kc + nc);
    if (lo < d->k_lo) lo = d->k_lo;
    if (hi > d->k_lo + d->n_f) hi = d->k_lo + d->n_f;
    const double *SA = d->psd + ((size_t)psd_row * 2 + 0) * (size_t)d->n_f;
    const double *SE = d->psd + ((size_t)psd_row * 2 + 1) * (size_t)d->n_f;
    double sum = 0.0;
    for (int64_t k = lo; k < hi; k++) {
        int64_t ib = k - kb, ic = k - kc, i = k - d->k_lo;
        double complex ba = bA[2 * ib] + I * bA[2 * ib + 1], ca = cA[2 * ic] + I * cA[2 * ic + 1];
        double complex be = bE[2 * ib] + I * bE[2 * ib + 1], ce = cE[2 * ic] + I * cE[2 * ic + 1];
        double ta = creal(conj(ba) * ca), te = creal(conj(be) * ce);
        if (d->psd_is_inverse) sum += ta * SA[i] + te * SE[i];
        else                   sum += ta / SA[i] + te / SE[i];
    }
    return 4.0 / cfg->Tobs * sum;
}

static int psd_row_of(const gbo_data *d, int w) {
    if (d->walker_psd) return d->walker_psd[w];
    return d->n_psd == 1 ? 0 : w;
}

/* residual of walker w viewed as a window over the whole stored band */
static const double *resid_ch(const gbo_data *d, int w, int ch) {
    return d->resid + (((size_t)w * 2 + (size_t)ch) * (size_t)d->n_f) * 2;
}

/* ---- O8  delta log-likelihood of one proposal row (Eq. 4, Eq. 5) ------- */
static int o8_row(const gbo_config *c, const gbo_data *d, const double *pnew, const double *pold,
                  int w, int mv, int N, double *dlnL, double *aux) {
    if (w < 0 || w >= d->n_walkers) return GBO_ERR_INVALID;
    int row = psd_row_of(d, w);
    const double *rA = resid_ch(d, w, 0), *rE = resid_ch(d, w, 1);
    double *buf = (double *)malloc(sizeof(double) * 8 * (size_t)N);
    double *aA = buf, *aE = buf + 2 * (size_t)N, *oA = buf + 4 * (size_t)N, *oE = buf + 6 * (size_t)N;
    int64_t ka = 0, ko = 0;
    int rc = GBO_OK;
    if (mv == GBO_ADD) {
        gbo_waveform(c, pnew, N, aA, aE, &ka);
        double aa = o7_inner(c, d, row, aA, aE, ka, N, aA, aE, ka, N);
        double ra = o7_inner(c, d, row, rA, rE, d->k_lo, (int)d->n_f, aA, aE, ka, N);
        *dlnL = ra - 0.5 * aa;                                  /* Eq. 4 with r = d - H */
        if (aux) { aux[0] = aa; aux[1] = ra; }
    } else if (mv == GBO_REMOVE) {
        gbo_waveform(c, pold, N, oA, oE, &ko);
        double oo = o7_inner(c, d, row, oA, oE, ko, N, oA, oE, ko, N);
        double ro = o7_inner(c, d, row, rA, rE, d->k_lo, (int)d->n_f, oA, oE, ko, N);
        *dlnL = -ro - 0.5 * oo;                                 /* Eq. 5 with a == 0     */
        if (aux) { aux[0] = oo; aux[1] = ro; }
    } else if (mv == GBO_SWAP) {
        gbo_waveform(c, pnew, N, aA, aE, &ka);
        gbo_waveform(c, pold, N, oA, oE, &ko);
        double aa = o7_inner(c, d, row, aA, aE, ka, N, aA, aE, ka, N);
        double oo = o7_inner(c, d, row, oA, oE, ko, N, oA, oE, ko, N);
        double ao = o7_inner(c, d, row, aA, aE, ka, N, oA, oE, ko, N);
        double ra = o7_inner(c, d, row, rA, rE, d->k_lo, (int)d->n_f, aA, aE, ka, N);
        double ro = o7_inner(c, d, row, rA, rE, d->k_lo, (int)d->n_f, oA, oE, ko, N);
        *dlnL = -0.5 * (aa + oo - 2.0 * ao - 2.0 * ra + 2.0 * ro);   /* Eq. 5 */
        if (aux) { aux[0] = aa; aux[1] = ra; }
    } else {
        rc = GBO_ERR_INVALID;
    }
    free(buf);
    return rc;
}

/* batched O8; proposals are evaluated independently against the same residual snapshot */
int gbo_delta_loglike(const gbo_config *c, const gbo_data *d, const double *params_new,
                      const double *params_old, const int32_t *walker_index, const int8_t *move,
                      int move_all, int N, const int32_t *n_bins, int64_t B,
                      double *dlnL_out, double *aux_out, int nthreads) {
    int bad = 0;
#pragma omp parallel for schedule(dynamic, 16) num_threads(nthreads > 0 ? nthreads : 1)
    for (int64_t b = 0; b < B; b++) {
        int mv = move ? move[b] : move_all;
        int Nb = n_bins ? n_bins[b] : N;
        if (!valid_N(Nb)) { bad = 1; continue; }
        const double *pn = params_new ? params_new + 8 * b : NULL;
        const double *po = params_old ? params_old + 8 * b : NULL;
        if ((mv != GBO_REMOVE && !pn) || (mv != GBO_ADD && !po)) { bad = 1; continue; }
        if (o8_row(c, d, pn, po, walker_index[b], mv, Nb, &dlnL_out[b], aux_out ? aux_out + 2 * b : NULL))
            bad = 1;
    }
    return bad ? GBO_ERR_INVALID : GBO_OK;
}

/* r[k] += sign * h[k] on the part of the window inside the stored band */
static void add_window(const gbo_data *d, int w, const double *hA, const double *hE, int64_t kh, int N, double sign) {
    double *rA = (double *)resid_ch(d, w, 0), *rE = (double *)resid_ch(d, w, 1);
    for (int j = 0; j < N; j++) {
        int64_t i = kh + j - d->k_lo;
        if (i < 0 || i >= d->n_f) continue;
        rA[2 * i] += sign * hA[2 * j]; rA[2 * i + 1] += sign * hA[2 * j + 1];
        rE[2 * i] += sign * hE[2 * j]; rE[2 * i + 1] += sign * hE[2 * j + 1];
    }
}

/* ---- O9  residual update (Alg. 1): rows applied in order b = 0..B-1 ------------
 * ADD: r -= a.  REMOVE: r += h.  SWAP: r += o, r -= a.  Rows of different walkers touch disjoint
 * memory, so handing whole walkers to different threads leaves every bit as in the sequential loop. */
int gbo_residual_update(const gbo_config *c, gbo_data *d, const double *params_new, const double *params_old,
                        const int32_t *walker_index, const int8_t *move, int move_all,
                        const uint8_t *accepted, int N, const int32_t *n_bins, int64_t B, int nthreads) {
    int bad = 0;
    for (int64_t b = 0; b < B; b++)
        if (walker_index[b] < 0 || walker_index[b] >= d->n_walkers) return GBO_ERR_INVALID;
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads > 0 ? nthreads : 1)
    for (int w = 0; w < d->n_walkers; w++) {
        for (int64_t b = 0; b < B; b++) {
            if (walker_index[b] != w || (accepted && !accepted[b])) continue;
            int mv = move ? move[b] : move_all;
            int Nb = n_bins ? n_bins[b] : N;
            if (!valid_N(Nb)) { bad = 1; continue; }
            double *h = (double *)malloc(sizeof(double) * 4 * (size_t)Nb), *hE = h + 2 * (size_t)Nb;
            int64_t kh;
            if (mv == GBO_REMOVE || mv == GBO_SWAP) {
                gbo_waveform(c, params_old + 8 * b, Nb, h, hE, &kh);
                add_window(d, w, h, hE, kh, Nb, +1.0);
            }
            if (mv == GBO_ADD || mv == GBO_SWAP) {
                gbo_waveform(c, params_new + 8 * b, Nb, h, hE, &kh);
                add_window(d, w, h, hE, kh, Nb, -1.0);
            }
            if (mv != GBO_ADD && mv != GBO_REMOVE && mv != GBO_SWAP) bad = 1;
            free(h);
        }
    }
    return bad ? GBO_ERR_INVALID : GBO_OK;
}

/* ---- the batched sweep step with its accept / reject decision (BASELINE config 5: "one waveform + delta lnL per source
 * per sweep ... then scatter-add of accepted deltas"; acceptance of Algorithm 1, with Eq. 13,
 * PAPER.md:197-202, in log form and the tempered likelihood of PAPER.md:674):
 *   1. delta lnL of EVERY row against the same residual snapshot (O8);
 *   2. row b is accepted iff  beta_b dlnL_b + logq_b >= logu_b   (logq NULL: 0, beta NULL: 1; a NaN dlnL is rejected);
 *   3. if apply: the accepted rows update the residual (O9), after all of step 1.
 * Written as exactly those three steps with the functions above. */
int gbo_delta_loglike_accept(const gbo_config *c, gbo_data *d, const double *params_new, const double *params_old,
                             const int32_t *walker_index, const int8_t *move, int move_all, int N, const int32_t *n_bins,
                             int64_t B, const double *logq, const double *logu, const double *beta, double *dlnL_out,
                             double *aux_out, uint8_t *accepted_out, int apply, int nthreads) {
    int rc = gbo_delta_loglike(c, d, params_new, params_old, walker_index, move, move_all, N, n_bins, B, dlnL_out, aux_out,
                               nthreads);
    if (rc) return rc;
    for (int64_t b = 0; b < B; b++) {
        double lhs = (beta ? beta[b] : 1.0) * dlnL_out[b] + (logq ? logq[b] : 0.0);
        accepted_out[b] = (uint8_t)(lhs >= logu[b] ? 1 : 0);
    }
    if (!apply) return GBO_OK;
    return gbo_residual_update(c, d, params_new, params_old, walker_index, move, move_all, accepted_out, N, n_bins, B,
                               nthreads);
}

/* <b|c> of two explicit windows against PSD row `psd_row` (exposed for pins P4-P6) */
double gbo_inner_windows(const gbo_config *c, const gbo_data *d, int psd_row,
                         const double *bA, const double *bE, int64_t kb, int nb,
                         const double *cA, const double *cE, int64_t kc, int nc) {
    return o7_inner(c, d, psd_row, bA, bE, kb, nb, cA, cE, kc, nc);
}

/* ---- normalised overlap of two sources (cataloging) -------------
 * O(a, c) = <a|c> / sqrt(<a|a> <c|c>) with Eq. 2 against PSD row psd_row[b], <a|c> over the bins common to
 * the two windows, every term over the stored band only.  The paper uses the overlap (threshold 0.9) and the
 * optimal SNR sqrt(<h|h>) (cut at 7) without printing the formula; this is the standard definition
 * (reading F4-a).  O = 0 when either norm vanishes (reading F4-b).  aux = (<a|a>, <c|c>).          */
int gbo_overlap(const gbo_config *c, const gbo_data *d, const double *params_a, const double *params_c,
                const int32_t *psd_row, int N, const int32_t *n_bins, int64_t B, double *overlap_out,
                double *aux_out, int nthreads) {
    int bad = 0;
#pragma omp parallel for schedule(dynamic, 16) num_threads(nthreads > 0 ? nthreads : 1)
    for (int64_t b = 0; b < B; b++) {
        int Nb = n_bins ? n_bins[b] : N;
        int row = psd_row ? psd_row[b] : 0;
        if (!valid_N(Nb) || row < 0 || row >= d->n_psd) { bad = 1; continue; }
        double *buf = (double *)malloc(sizeof(double) * 8 * (size_t)Nb);
        double *aA = buf, *aE = buf + 2 * (size_t)Nb, *cA = buf + 4 * (size_t)Nb, *cE = buf + 6 * (size_t)Nb;
        int64_t ka, kc;
        gbo_waveform(c, params_a + 8 * b, Nb, aA, aE, &ka);
        gbo_waveform(c, params_c + 8 * b, Nb, cA, cE, &kc);
        double aa = o7_inner(c, d, row, aA, aE, ka, Nb, aA, aE, ka, Nb);
        double cc = o7_inner(c, d, row, cA, cE, kc, Nb, cA, cE, kc, Nb);
        double ac = o7_inner(c, d, row, aA, aE, ka, Nb, cA, cE, kc, Nb);
        overlap_out[b] = (aa > 0.0 && cc > 0.0) ? ac / sqrt(aa * cc) : 0.0;
        if (aux_out) { aux_out[2 * b] = aa; aux_out[2 * b + 1] = cc; }
        free(buf);
    }
    return bad ? GBO_ERR_INVALID : GBO_OK;
}

/* ---- Algorithm 1: sequential proposals of one band against a staged residual --------
 * One task = one band j = (t, w, b): the residual r' of walker `walker` on the staged bins
 * [k_first, k_first + n_stage) (the paper's sub-bands b-1, b, b+1; reading F1-a: the caller's
 * per-(t,w) residual already has the current sources subtracted, r = d - H), the band's n_src sources
 * params[src_begin ..], and n_prop proposals applied IN ORDER: proposal p replaces
 * source k_p by theta'_p; delta lnL by Eq. 5 with every inner product restricted to the
 * staged bins (and the stored band); accepted iff beta * dlnL + logq_p >= logu_p (Eq. 13
 * in log form with the tempered likelihood of PAPER.md:674; logq_p = log prior/proposal ratio and logu_p =
 * log of the uniform draw are inputs: the random numbers of the method are passed in).  On acceptance
 * theta_j[k] <- theta', r' <- r' + h(theta_k) - h(theta'_k).  If write_back, the net
 * change of r' is added to the walker's stored residual at the end.  Tasks are processed
 * one after the other in task order.
 * Odd/even cold-chain buffers (Fig. 4; row f3), flags bits 1 and 2:
 *   bit 1 (2): r' is formed ONLINE: the staged row holds the data minus the cold-chain sources of the OTHER
 *              parity only, and the band's own current sources are subtracted while staging
 *              ("We subtract from the buffer residual the waveforms contained in (w, t, b)", :360);
 *   bit 2 (4): the write-back goes to row `write_walker` (the buffer of the band's own parity, :362) instead
 *              of the staged row.                                                                       */
typedef struct {
    int32_t walker, n_src, src_begin, n_prop, prop_begin, n_stage;
    int64_t k_first;
    int32_t flags, write_walker;     /* flags: 1 write back, 2 subtract current sources, 4 write to write_walker */
    double beta;
} gbo_band_task;

/* ---- proposal generation inside Algorithm 1 ("k <- randint(0, g_j)", "theta'_k <- Make Proposal
 * on theta"; group stretch of App. B; stretch move Eq. 14) --------------------
 * The random numbers come from the counter-based generator Philox4x32-10 (Salmon et al. 2011), written out below and
 * pinned to its published known-answer vectors.  Key = the 64-bit seed; counter = (global proposal row, 0, block, sweep):
 * a proposal's numbers depend on nothing but (seed, sweep, its row in the proposal arrays), not on the order in which
 * tasks are processed.  Block 0 gives k, the friend and z; block 1 gives the uniform of the accept / reject step.
 * Readings (paper-silent points; F1-h..F1-m):
 *   randint          k = floor(r g_j / 2^32) for a 32-bit word r
 *   uniforms         u = (a + 1/2) 2^-52, a = the top 26 bits of two words: 0 < u < 1
 *   stationary group rows of 8 parameters sorted by f0 ascending ("sorting this large set of templates by
 *                    frequency"); the n_friends rows closest in f0 to the CURRENT theta_k are a run of consecutive rows
 *                    (equal distances: the run with the lower rows); the auxiliary point is friend
 *                    floor(r n_friends / 2^32) of that run (":576 draws uniformly")
 *   stretch density  g(z) ~ 1/sqrt(z) on [1/a, a] (ref. [59] of the paper), z = ((a - 1) u + 1)^2 / a
 *   move             theta' = theta_aux + z (theta_k - theta_aux) on all D = 8 coordinates of the parameter row (Eq. 14),
 *                    proposal-density factor z^(D-1): logq = 7 ln z
 *   periodic         coordinates flagged periodic are wrapped into [lo, hi): x - (hi - lo) floor((x - lo) / (hi - lo))
 *   prior            uniform on the box [lo, hi] per coordinate (Eq. 13's prior ratio is 1 inside, 0 outside): a proposal
 *                    outside the box is rejected without a likelihood evaluation (delta lnL reported as NaN); the same for a
 *                    proposal whose window leaves the staged bins (applied in the sweep loop below)       */
typedef struct {
    uint64_t seed;
    uint32_t sweep;
    int32_t n_friends;
    const double *group;      /* [n_group][8], sorted by f0 (column 1) ascending */
    int64_t n_group;
    double stretch_a;
    double lo[8], hi[8];
    int32_t periodic[8];
} gbo_stretch;

void gbo_philox4x32_10(const uint32_t ctr_in[4], const uint32_t key_in[2], uint32_t out[4]) {
    uint32_t c[4] = {ctr_in[0], ctr_in[1], ctr_in[2], ctr_in[3]};
    uint32_t k[2] = {key_in[0], key_in[1]};
    for (int round = 0; round < 10; round++) {
        if (round > 0) { k[0] += 0x9E3779B9u; k[1] += 0xBB67AE85u; }      /* Weyl sequence of the key */
        uint64_t p0 = (uint64_t)0xD2511F53u * c[0];
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c[2];
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c[1] ^ k[0], n1 = lo1, n2 = hi0 ^ c[3] ^ k[1], n3 = lo0;
        c[0] = n0; c[1] = n1; c[2] = n2; c[3] = n3;
    }
    for (int i = 0; i < 4; i++) out[i] = c[i];
}

static void proposal_words(const gbo_stretch *g, int64_t row, uint32_t block, uint32_t out[4]) {
    uint32_t ctr[4] = {(uint32_t)row, 0u, block, g->sweep};
    uint32_t key[2] = {(uint32_t)(g->seed & 0xffffffffu), (uint32_t)(g->seed >> 32)};
    gbo_philox4x32_10(ctr, key, out);
}

double gbo_uniform52(uint32_t w0, uint32_t w1) {                /* 0 < u < 1, 52 random bits */
    double a = (double)(w0 >> 6) * 67108864.0 + (double)(w1 >> 6);
    return (a + 0.5) * (1.0 / 4503599627370496.0);
}

int32_t gbo_randint(uint32_t w, int32_t n) { return (int32_t)(((uint64_t)w * (uint64_t)n) >> 32); }

double gbo_stretch_z(double u, double a) {                       /* inverse CDF of g(z) ~ z^(-1/2) on [1/a, a] */
    double t = (a - 1.0) * u + 1.0;
    return t * t / a;
}

/* row of the j-th of the n_friends group points closest in f0 to f.  The table is sorted by f0, so the
 * closest n_friends rows are a run of consecutive rows [s, s + n_friends): the first s at which trading row s for row
 * s + n_friends would not bring the run closer to f, found by trying every s in turn; the j-th friend is row s + j.
 * (Equal distances: the run with the lower rows.)                                                                       */
int64_t gbo_friend_row(const double *group, int64_t n_group, int32_t n_friends, double f, int32_t j) {
    int64_t nf = n_friends < n_group ? n_friends : n_group;
    int64_t s = 0;
    while (s < n_group - nf && f - group[8 * s + P_F0] > group[8 * (s + nf) + P_F0] - f) s++;
    return s + j;
}

/* "theta'_k <- Make Proposal on theta" for global proposal row `row` of a band with g_j current sources
 * theta[g_j][8].  Returns 1 if theta' lies inside the prior box, else 0.                                            */
int gbo_make_proposal(const gbo_stretch *g, int64_t row, const double *theta, int32_t g_j, int32_t *k_out,
                      double *theta_prop, double *logq, double *logu) {
    uint32_t w0[4], w1[4];
    proposal_words(g, row, 0u, w0);
    proposal_words(g, row, 1u, w1);
    int32_t k = gbo_randint(w0[0], g_j);                           /* k <- randint(0, g_j) */
    const double *theta_k = theta + 8 * (size_t)k;
    int64_t nf = g->n_friends < g->n_group ? g->n_friends : g->n_group;
    int32_t j = gbo_randint(w0[1], (int32_t)nf);
    const double *aux = g->group + 8 * gbo_friend_row(g->group, g->n_group, g->n_friends, theta_k[P_F0], j);
    double z = gbo_stretch_z(gbo_uniform52(w0[2], w0[3]), g->stretch_a);
    int inside = 1;
    for (int cdx = 0; cdx < 8; cdx++) {
        double x = aux[cdx] + z * (theta_k[cdx] - aux[cdx]);      /* Eq. 14 */
        if (g->periodic[cdx]) {
            double period = g->hi[cdx] - g->lo[cdx];
            x = x - period * floor((x - g->lo[cdx]) / period);
        }
        if (!(x >= g->lo[cdx] && x <= g->hi[cdx])) inside = 0;
        theta_prop[cdx] = x;
    }
    *k_out = k;
    *logq = 7.0 * log(z);                                          /* z^(D-1), D = 8 */
    *logu = log(gbo_uniform52(w1[0], w1[1]));
    return inside;
}

static int band_sweep_impl(const gbo_config *c, gbo_data *d, const gbo_band_task *tasks, int64_t n_tasks, int N,
                           double *params, const int32_t *prop_k, const double *prop_params, const double *prop_logq,
                           const double *prop_logu, uint8_t *accepted_out, double *dlnL_out,
                           const gbo_stretch *gen, int32_t *k_gen, double *params_gen, double *logq_gen, double *logu_gen) {
    if (!valid_N(N)) return GBO_ERR_INVALID;
    double *h = (double *)malloc(sizeof(double) * 8 * (size_t)N);
    double *oA = h, *oE = h + 2 * (size_t)N, *aA = h + 4 * (size_t)N, *aE = h + 6 * (size_t)N;
    for (int64_t it = 0; it < n_tasks; it++) {
        const gbo_band_task *t = &tasks[it];
        if (t->walker < 0 || t->walker >= d->n_walkers || t->n_stage < 0) { free(h); return GBO_ERR_INVALID; }
        /* staged bins that are stored: global bins [lo, hi) */
        int64_t lo = t->k_first > d->k_lo ? t->k_first : d->k_lo;
        int64_t hi = t->k_first + t->n_stage < d->k_lo + d->n_f ? t->k_first + t->n_stage : d->k_lo + d->n_f;
        int64_t n = hi > lo ? hi - lo : 0;
        /* r' and the PSD of the walker on those bins, as a one-walker data view */
        double *rv = (double *)malloc(sizeof(double) * 4 * (size_t)(n > 0 ? n : 1));
        double *r0 = (double *)malloc(sizeof(double) * 4 * (size_t)(n > 0 ? n : 1));
        double *sv = (double *)malloc(sizeof(double) * 2 * (size_t)(n > 0 ? n : 1));
        int row = psd_row_of(d, t->walker);
        for (int ch = 0; ch < 2; ch++) {
            const double *r = resid_ch(d, t->walker, ch) + 2 * (lo - d->k_lo);
            const double *S = d->psd + ((size_t)row * 2 + (size_t)ch) * (size_t)d->n_f + (lo - d->k_lo);
            for (int64_t i = 0; i < n; i++) {
                rv[2 * ((size_t)ch * n + i)] = r[2 * i];
                rv[2 * ((size_t)ch * n + i) + 1] = r[2 * i + 1];
                sv[(size_t)ch * n + i] = S[i];
            }
        }
        gbo_data v = {rv, sv, NULL, lo, n, 1, 1, d->psd_is_inverse};
        if ((t->flags & 2) && n > 0) {                     /* r' <- r' - sum of the band's current sources (:360) */
            for (int sidx = 0; sidx < t->n_src; sidx++) {
                int64_t kh;
                gbo_waveform(c, params + 8 * ((size_t)t->src_begin + sidx), N, oA, oE, &kh);
                add_window(&v, 0, oA, oE, kh, N, -1.0);
            }
        }
        memcpy(r0, rv, sizeof(double) * 4 * (size_t)n);
        for (int p = 0; p < t->n_prop && n > 0; p++) {
            int64_t ip = t->prop_begin + p;
            int k;
            const double *theta_p;
            double lq, lu;
            if (gen) {                             /* k <- randint(0, g_j); theta'_k <- Make Proposal */
                if (t->n_src <= 0) { free(rv); free(r0); free(sv); free(h); return GBO_ERR_INVALID; }
                int32_t kk;
                int inside = gbo_make_proposal(gen, ip, params + 8 * (size_t)t->src_begin, t->n_src, &kk,
                                               params_gen + 8 * ip, &logq_gen[ip], &logu_gen[ip]);
                k_gen[ip] = kk;
                /* "We allow samples to go halfway into neighboring bands": with a window as wide as a
                 * sub-band that is exactly the condition that the window of theta' stays on the staged sub-bands b-1, b, b+1;
                 * beyond that the prior is zero (reading F1-n)                                                */
                {
                    double prod = params_gen[8 * ip + P_F0] * c->Tobs;
                    int64_t kmin_p = (int64_t)floor(prod + 0.5) - N / 2;
                    if (kmin_p < t->k_first || kmin_p + N > t->k_first + t->n_stage) inside = 0;
                }
                if (!inside) {                     /* zero prior: rejected, no likelihood evaluation */
                    dlnL_out[ip] = NAN;
                    accepted_out[ip] = 0;
                    continue;
                }
                k = kk; theta_p = params_gen + 8 * ip; lq = logq_gen[ip]; lu = logu_gen[ip];
            } else {
                k = prop_k[ip]; theta_p = prop_params + 8 * ip; lq = prop_logq[ip]; lu = prop_logu[ip];
            }
            if (k < 0 || k >= t->n_src) { free(rv); free(r0); free(sv); free(h); return GBO_ERR_INVALID; }
            double *theta_k = params + 8 * ((size_t)t->src_begin + k);
            double dl = 0.0;
            o8_row(c, &v, theta_p, theta_k, 0, GBO_SWAP, N, &dl, NULL);            /* Eq. 5 against r' */
            int acc = t->beta * dl + lq >= lu;
            dlnL_out[ip] = dl;
            accepted_out[ip] = (uint8_t)acc;
            if (acc) {
                int64_t ko, ka;
                gbo_waveform(c, theta_k, N, oA, oE, &ko);
                gbo_waveform(c, theta_p, N, aA, aE, &ka);
                add_window(&v, 0, oA, oE, ko, N, +1.0);                             /* r' += h(theta_k)  */
                add_window(&v, 0, aA, aE, ka, N, -1.0);                             /* r' -= h(theta'_k) */
                memcpy(theta_k, theta_p, sizeof(double) * 8);
            }
        }
        for (int p = 0; p < t->n_prop && n <= 0; p++) {   /* nothing staged: every dlnL is 0 */
            int64_t ip = t->prop_begin + p;
            if (gen) { free(rv); free(r0); free(sv); free(h); return GBO_ERR_INVALID; }   /* generating needs staged bins */
            int acc = prop_logq[ip] >= prop_logu[ip];
            dlnL_out[ip] = 0.0;
            accepted_out[ip] = (uint8_t)acc;
            if (acc) memcpy(params + 8 * ((size_t)t->src_begin + prop_k[ip]), prop_params + 8 * ip, sizeof(double) * 8);
        }
        if (t->flags & 1) {
            int wrow = (t->flags & 4) ? t->write_walker : t->walker;
            if (wrow < 0 || wrow >= d->n_walkers) { free(rv); free(r0); free(sv); free(h); return GBO_ERR_INVALID; }
            for (int ch = 0; ch < 2; ch++) {
                double *r = (double *)resid_ch(d, wrow, ch) + 2 * (lo - d->k_lo);
                for (int64_t i = 0; i < 2 * n; i++) r[i] += rv[2 * (size_t)ch * n + i] - r0[2 * (size_t)ch * n + i];
            }
        }
        free(rv); free(r0); free(sv);
    }
    free(h);
    return GBO_OK;
}

/* Algorithm 1 with k, theta', logq and logu given by the caller (reading F1-b) */
int gbo_band_sweep(const gbo_config *c, gbo_data *d, const gbo_band_task *tasks, int64_t n_tasks, int N,
                   double *params, const int32_t *prop_k, const double *prop_params, const double *prop_logq,
                   const double *prop_logu, uint8_t *accepted_out, double *dlnL_out) {
    return band_sweep_impl(c, d, tasks, n_tasks, N, params, prop_k, prop_params, prop_logq, prop_logu, accepted_out,
                           dlnL_out, NULL, NULL, NULL, NULL, NULL);
}

/* Algorithm 1 as printed: the proposal step runs inside the loop, from the CURRENT theta_k.
 * k_out, params_out [.][8], logq_out, logu_out receive what was generated for every proposal row.            */
int gbo_band_sweep_generate(const gbo_config *c, gbo_data *d, const gbo_band_task *tasks, int64_t n_tasks, int N,
                            double *params, const gbo_stretch *gen, int32_t *k_out, double *params_out,
                            double *logq_out, double *logu_out, uint8_t *accepted_out, double *dlnL_out) {
    if (!gen || !gen->group || gen->n_group < 1 || gen->n_friends < 1 || !(gen->stretch_a > 1.0)) return GBO_ERR_INVALID;
    return band_sweep_impl(c, d, tasks, n_tasks, N, params, NULL, NULL, NULL, NULL, accepted_out, dlnL_out,
                           gen, k_out, params_out, logq_out, logu_out);
}

/* ---- Algorithm 2 (Eq. D2): temperature swaps of one sub-band ------------
 * One task = one sub-band b with a ladder of n_t chains.  Chain t has a residual row chain_walker[t] (the
 * paper's permuted walker p[t]; r = d - H of that chain, reading F1-a), an inverse temperature
 * chain_beta[t] and the set of the band's sources it currently holds, params rows
 * [chain_set_begin[t], + chain_set_n[t]).  From the hottest pair down (t = n_t-1 .. 1) chains
 * i = t and j = t-1 propose to exchange their sets S_i <-> S_j.  With delta = sum_{S_i} h - sum_{S_j} h on the
 * staged bins (both residuals change by +-delta if the sets are exchanged),
 *     D_i = lnL_i(S_j) - lnL_i(S_i) = -1/2 <delta|delta>_i - <r_i|delta>_i
 *     D_j = lnL_j(S_i) - lnL_j(S_j) = -1/2 <delta|delta>_j + <r_j|delta>_j       (Eq. 1-2 with each chain's PSD row)
 * and the swap is accepted iff beta_i D_i + beta_j D_j >= logu[t]   (Eq. D2 in log form; logu is an input).
 * If accepted the sets are exchanged, r_i += delta, r_j -= delta on the staged bins of every
 * chain whose write_back flag is set (the paper stores only the cold chain, :652-658; here every chain owns a
 * residual), and the next pair sees the new holder of chain t-1.  Outputs per chain entry t: accepted[t] and
 * dlnl[t] = (D_i, D_j) of the pair (t, t-1) (entry 0 unused), perm[t] = the chain whose INITIAL set ends in t. */
/* Odd/even cold-chain buffers (Algorithm 2 as printed): with bit 2 of write_back the
 * stored row of a chain's walker holds NONE of the band's own sources (it is the opposite-parity cold-chain buffer, which
 * carries only the leakage of the neighbours), so each chain's residual is formed first, r_t = row(p[t]) - sum_{S_t} h
 * over the set the chain holds ("r' <- r_(0,w,b-1) + r_(0,w,b+1) - sum h"), and only an exchange with the
 * cold chain (t - 1 = 0) is written, as -delta into row write_walker, the cold chain's buffer of the band's own parity
 * ("if t = 1 ... update cold-chain residual").                                                        */
typedef struct {
    int32_t n_t, chain_begin, n_stage, write_back;   /* write_back: bit 1 = write accepted exchanges, bit 2 = odd/even mode */
    int64_t k_first;
    int32_t write_walker, reserved;
} gbo_temper_task;

int gbo_temper_sweep(const gbo_config *c, gbo_data *d, const gbo_temper_task *tasks, int64_t n_tasks, int N,
                     const double *params, const int32_t *chain_walker, const double *chain_beta,
                     const int32_t *chain_set_begin, const int32_t *chain_set_n, const double *chain_logu,
                     int32_t *perm_out, uint8_t *accepted_out, double *dlnl_out) {
    if (!valid_N(N)) return GBO_ERR_INVALID;
    double *hA = (double *)malloc(sizeof(double) * 4 * (size_t)N), *hE = hA + 2 * (size_t)N;
    for (int64_t it = 0; it < n_tasks; it++) {
        const gbo_temper_task *t = &tasks[it];
        int64_t lo = t->k_first > d->k_lo ? t->k_first : d->k_lo;
        int64_t hi = t->k_first + t->n_stage < d->k_lo + d->n_f ? t->k_first + t->n_stage : d->k_lo + d->n_f;
        int64_t n = hi > lo ? hi - lo : 0;
        double complex *dl = (double complex *)malloc(sizeof(double complex) * 2 * (size_t)(n > 0 ? n : 1));
        double complex *hs = (double complex *)malloc(sizeof(double complex) * 4 * (size_t)(n > 0 ? n : 1));   /* H_i, H_j */
        const int oddeven = (t->write_back & 2) != 0;
        int *holder = (int *)malloc(sizeof(int) * (size_t)(t->n_t > 0 ? t->n_t : 1));   /* whose initial set chain t holds */
        for (int q = 0; q < t->n_t; q++) { holder[q] = q; perm_out[t->chain_begin + q] = q; accepted_out[t->chain_begin + q] = 0;
                                           dlnl_out[2 * (t->chain_begin + q)] = dlnl_out[2 * (t->chain_begin + q) + 1] = 0.0; }
        for (int q = t->n_t - 1; q >= 1; q--) {
            int ci = t->chain_begin + q, cj = ci - 1;
            int wi = chain_walker[ci], wj = chain_walker[cj];
            if (wi < 0 || wi >= d->n_walkers || wj < 0 || wj >= d->n_walkers) { free(dl); free(hs); free(holder); free(hA); return GBO_ERR_INVALID; }
            /* delta = sum over the set chain i holds - sum over the set chain j holds, on the staged stored bins */
            for (int64_t x = 0; x < 2 * n; x++) dl[x] = 0.0;
            for (int64_t x = 0; x < 4 * n; x++) hs[x] = 0.0;
            for (int side = 0; side < 2; side++) {
                int src = t->chain_begin + holder[side == 0 ? q : q - 1];
                double sign = side == 0 ? +1.0 : -1.0;
                double complex *H = hs + (size_t)side * 2 * n;          /* the sum of the set this chain holds */
                for (int sidx = 0; sidx < chain_set_n[src]; sidx++) {
                    int64_t kh;
                    gbo_waveform(c, params + 8 * ((size_t)chain_set_begin[src] + sidx), N, hA, hE, &kh);
                    for (int jb = 0; jb < N; jb++) {
                        int64_t k = kh + jb;
                        if (k < lo || k >= hi) continue;
                        dl[k - lo] += sign * (hA[2 * jb] + I * hA[2 * jb + 1]);
                        dl[n + k - lo] += sign * (hE[2 * jb] + I * hE[2 * jb + 1]);
                        H[k - lo] += hA[2 * jb] + I * hA[2 * jb + 1];
                        H[n + k - lo] += hE[2 * jb] + I * hE[2 * jb + 1];
                    }
                }
            }
            double D[2];
            for (int side = 0; side < 2; side++) {                 /* side 0: chain i (+<r|delta> enters with -), side 1: chain j */
                int w = side == 0 ? wi : wj, row = psd_row_of(d, w);
                double dd = 0.0, rd = 0.0;
                for (int ch = 0; ch < 2; ch++) {
                    const double *r = resid_ch(d, w, ch) + 2 * (lo - d->k_lo);
                    const double *S = d->psd + ((size_t)row * 2 + (size_t)ch) * (size_t)d->n_f + (lo - d->k_lo);
                    for (int64_t x = 0; x < n; x++) {
                        double complex de = dl[(size_t)ch * n + x], rr = r[2 * x] + I * r[2 * x + 1];
                        if (oddeven) rr -= hs[(size_t)side * 2 * n + (size_t)ch * n + x];   /* r_t = row - sum_{S_t} h */
                        double wgt = d->psd_is_inverse ? S[x] : 1.0 / S[x];
                        dd += wgt * creal(conj(de) * de);
                        rd += wgt * creal(conj(rr) * de);
                    }
                }
                dd *= 4.0 / c->Tobs; rd *= 4.0 / c->Tobs;
                D[side] = side == 0 ? -0.5 * dd - rd : -0.5 * dd + rd;
            }
            int acc = chain_beta[ci] * D[0] + chain_beta[cj] * D[1] >= chain_logu[ci];
            accepted_out[ci] = (uint8_t)acc;
            dlnl_out[2 * ci] = D[0]; dlnl_out[2 * ci + 1] = D[1];
            if (acc) {
                int tmp = holder[q]; holder[q] = holder[q - 1]; holder[q - 1] = tmp;
                if (oddeven) {
                    if ((t->write_back & 1) && q - 1 == 0) {       /* the cold chain now holds S_i: its own-parity buffer -= delta */
                        if (t->write_walker < 0 || t->write_walker >= d->n_walkers) { free(dl); free(hs); free(holder); free(hA); return GBO_ERR_INVALID; }
                        for (int ch = 0; ch < 2; ch++) {
                            double *rw = (double *)resid_ch(d, t->write_walker, ch) + 2 * (lo - d->k_lo);
                            for (int64_t x = 0; x < n; x++) {
                                double complex de = dl[(size_t)ch * n + x];
                                rw[2 * x] -= creal(de); rw[2 * x + 1] -= cimag(de);
                            }
                        }
                    }
                } else if (t->write_back & 1) {
                    for (int ch = 0; ch < 2; ch++) {
                        double *ri = (double *)resid_ch(d, wi, ch) + 2 * (lo - d->k_lo);
                        double *rj = (double *)resid_ch(d, wj, ch) + 2 * (lo - d->k_lo);
                        for (int64_t x = 0; x < n; x++) {
                            double complex de = dl[(size_t)ch * n + x];
                            ri[2 * x] += creal(de); ri[2 * x + 1] += cimag(de);
                            rj[2 * x] -= creal(de); rj[2 * x + 1] -= cimag(de);
                        }
                    }
                }
            }
        }
        for (int q = 0; q < t->n_t; q++) perm_out[t->chain_begin + q] = holder[q];
        free(dl); free(hs); free(holder);
    }
    free(hA);
    return GBO_OK;
}

/* orbit positions at time t, row-major [3][3] (exposed for the orbit pin) */
void gbo_orbits(const gbo_config *c, double t, double *x_out) {
    double x[3][3];
    o2_orbits(c, t, x);
    memcpy(x_out, x, sizeof(x));
}

int gbo_max_threads(void) {
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    return omp_get_max_threads();
#else
    return 1;
#endif
}
