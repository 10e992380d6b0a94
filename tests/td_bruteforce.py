"""Independent time-domain brute force used to PIN the oracle (tests only; numpy; shares nothing with
oracle/gb_oracle.c or with the CUDA path).

It evaluates the *real* TDI-1.5 Michelson observables from their definition:
  h(xi)      = h_plus(xi) eps_plus + h_cross(xi) eps_cross                     (rank-2 tensor)
  H_rs(xi)   = n_rs . h(xi) . n_rs
  y_rs(t)    = [H_rs(t - tau - k.x_s/c) - H_rs(t - k.x_r/c)] / (2 (1 - k.n_rs))   (one-way Doppler link)
  X(t)       = y13 + D y31 + D^2 y12 + D^3 y21 - [y12 + D y21 + D^2 y13 + D^3 y31]  (delay D = tau)
  A = (Z - X)/sqrt2, E = (X - 2Y + Z)/sqrt6                                      (Eq. 6)
with no complex envelope, no sinc/transfer-function algebra and no delay phasors.  The strain follows
DESIGN.md readings S3/S7/S8: Phi(xi) = 2 pi f0 xi + pi fdot xi^2 + phi0, amplitude factor
1 + (2/3)(fdot/f0) xi, h_plus = amp (1 + cos^2 iota) cos Phi, h_cross = -2 amp cos(iota) sin Phi.
"""
import numpy as np

C_LIGHT = 299792458.0


def orbits(cfg, t):
    """Spacecraft positions [3][..., 3] at times t -- DESIGN.md reading S2 (first order in e)."""
    t = np.asarray(t, dtype=np.float64)
    al = 2.0 * np.pi * t / cfg.year + cfg.kappa
    e = cfg.armlength / (2.0 * np.sqrt(3.0) * cfg.au)
    out = []
    for i in range(3):
        b = 2.0 * np.pi * i / 3.0 + cfg.lambda0
        x = cfg.au * np.cos(al) + cfg.au * e * (np.sin(al) * np.cos(al) * np.sin(b) - (1 + np.sin(al) ** 2) * np.cos(b))
        y = cfg.au * np.sin(al) + cfg.au * e * (np.sin(al) * np.cos(al) * np.cos(b) - (1 + np.cos(al) ** 2) * np.sin(b))
        z = -np.sqrt(3.0) * cfg.au * e * np.cos(al - b)
        out.append(np.stack([x, y, z], -1))
    return out


def source_frame(p):
    amp, f0, fd, phi0, ci, psi, lam, sb = p
    cb = np.sqrt(1.0 - sb * sb)
    k = -np.array([cb * np.cos(lam), cb * np.sin(lam), sb])
    u = np.array([sb * np.cos(lam), sb * np.sin(lam), -cb])
    v = np.array([np.sin(lam), -np.cos(lam), 0.0])
    ep = np.outer(u, u) - np.outer(v, v)
    ec = np.outer(u, v) + np.outer(v, u)
    Ep = np.cos(2 * psi) * ep - np.sin(2 * psi) * ec
    Ec = np.sin(2 * psi) * ep + np.cos(2 * psi) * ec
    return k, u, v, Ep, Ec


def carrier_split(cfg, p):
    """q = round(f0 T) and delta = f0 T - q evaluated in extended precision (independent of the oracle's fma)."""
    f0 = np.longdouble(p[1])
    T = np.longdouble(cfg.Tobs)
    q = int(np.floor(f0 * T + np.longdouble(0.5)))
    return q, float(f0 * T - np.longdouble(q))


def real_AE(cfg, p, t, cyc_t, phi0_shift=0.0, moving=False):
    """Real A(t), E(t) at times t.  cyc_t = f0 * t in cycles, supplied by the caller reduced modulo 1
    where possible so that the carrier phase keeps full precision.  moving=False freezes the geometry
    at t (pin P1); moving=True re-evaluates positions at each reception / emission time (pin P3)."""
    amp, f0, fd, phi0, ci, psi, lam, sb = p
    phi0 = phi0 + phi0_shift
    L = cfg.armlength
    tau = L / C_LIGHT
    k, u, v, Ep, Ec = source_frame(p)
    Apl = amp * (1.0 + ci * ci)
    Acr = -2.0 * amp * ci
    X0 = orbits(cfg, t)

    def H(nvec, s):
        """n.h(xi).n at retarded time xi = t - s."""
        xi = t - s
        Phi = 2.0 * np.pi * (cyc_t - f0 * s) + np.pi * fd * xi * xi + phi0
        a = 1.0 + (2.0 / 3.0) * (fd / f0) * xi
        dp = ((nvec @ Ep) * nvec).sum(-1)                 # n . eps_plus . n
        dc = ((nvec @ Ec) * nvec).sum(-1)                 # n . eps_cross . n
        return a * (Apl * np.cos(Phi) * dp + Acr * np.sin(Phi) * dc)

    def y(r, s, m):
        """y_rs evaluated at t - m tau."""
        if moving:
            xr = orbits(cfg, t - m * tau)[r]
            xs = orbits(cfg, t - m * tau - tau)[s]
        else:
            xr, xs = X0[r], X0[s]
        nrs = (xr - xs) / L
        kap = nrs @ k
        return (H(nrs, m * tau + tau + xs @ k / C_LIGHT) - H(nrs, m * tau + xr @ k / C_LIGHT)) / (2.0 * (1.0 - kap))

    def michelson(i1, i2, i3):
        return (y(i1, i3, 0) + y(i3, i1, 1) + y(i1, i2, 2) + y(i2, i1, 3)) \
             - (y(i1, i2, 0) + y(i2, i1, 1) + y(i1, i3, 2) + y(i3, i1, 3))

    Xx, Yy, Zz = michelson(0, 1, 2), michelson(1, 2, 0), michelson(2, 0, 1)
    return (Zz - Xx) / np.sqrt(2.0), (Xx - 2.0 * Yy + Zz) / np.sqrt(6.0)


def coarse_window(cfg, p, N, moving=False):
    """Pin P1 / P3: analytic signal at the N coarse times -> heterodyne by bin q -> DFT -> T/(2N).
    Returns (A[N], E[N], kmin) in the oracle's bin convention."""
    q, delta = carrier_split(cfg, p)
    n = np.arange(N)
    t = n * cfg.Tobs / N
    cyc = ((q * n) % N) / N + delta * n / N              # f0 t_n modulo 1 (integer split)
    A0, E0 = real_AE(cfg, p, t, cyc, 0.0, moving)
    A1, E1 = real_AE(cfg, p, t, cyc, np.pi / 2.0, moving)
    het = np.exp(-2j * np.pi * ((q * n) % N) / N)
    za, ze = (A0 - 1j * A1) * het, (E0 - 1j * E1) * het
    scale = cfg.Tobs / (2.0 * N)
    Fa = np.fft.fftshift(np.fft.fft(za)) * scale
    Fe = np.fft.fftshift(np.fft.fft(ze)) * scale
    return Fa, Fe, q - N // 2


def full_rate_window(cfg, p, N, moving=False, chunk=1 << 20):
    """Pin P2: real signal at all M = T/dt samples, true dt * rfft, cut to the oracle's window."""
    M = int(round(cfg.Tobs / cfg.dt))
    q, _ = carrier_split(cfg, p)
    A = np.empty(M)
    E = np.empty(M)
    f0 = np.longdouble(p[1])
    for s in range(0, M, chunk):
        m = np.arange(s, min(M, s + chunk))
        t = m * cfg.dt
        cyc = np.asarray((f0 * np.asarray(t, dtype=np.longdouble)) % 1, dtype=np.float64)
        A[m], E[m] = real_AE(cfg, p, t, cyc, 0.0, moving)
    kmin = q - N // 2
    FA = cfg.dt * np.fft.rfft(A)
    FE = cfg.dt * np.fft.rfft(E)
    return FA[kmin:kmin + N], FE[kmin:kmin + N], kmin, FA, FE
