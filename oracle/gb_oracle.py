"""ctypes wrapper around oracle/gb_oracle.c (the CPU oracle).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  The product package never imports this module.

All arithmetic of the method lives in gb_oracle.c; this file only marshals numpy arrays.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gb_oracle.c")
_LIB = os.path.join(_HERE, "libgb_oracle.so")

ADD, REMOVE, SWAP = 0, 1, 2


def build(force: bool = False) -> str:
    """Compile gb_oracle.c -> libgb_oracle.so (gcc, -O2, no FMA contraction, OpenMP)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-std=c11", "-O2", "-ffp-contract=off", "-fopenmp", "-Wall", "-Wextra",
               "-shared", "-fPIC", _SRC, "-o", _LIB, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class _Config(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("Tobs", "dt", "armlength", "au", "year", "kappa", "lambda0")]


class _Data(C.Structure):
    _fields_ = [("resid", C.c_void_p), ("psd", C.c_void_p), ("walker_psd", C.c_void_p),
                ("k_lo", C.c_int64), ("n_f", C.c_int64),
                ("n_walkers", C.c_int32), ("n_psd", C.c_int32), ("psd_is_inverse", C.c_int32)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.gbo_inner_windows.restype = C.c_double
    return _lib


@dataclass
class Config:
    Tobs: float = 31457280.0
    dt: float = 5.0
    armlength: float = 2.5e9
    au: float = 1.495978707e11
    year: float = 31558149.763545603
    kappa: float = 0.0
    lambda0: float = 0.0

    def c(self) -> _Config:
        return _Config(self.Tobs, self.dt, self.armlength, self.au, self.year, self.kappa, self.lambda0)


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def max_threads() -> int:
    return int(lib().gbo_max_threads())


class Data:
    """Host residual / PSD view.  resid: complex128 [n_walkers, 2, n_f] (modified in place by
    residual_update); psd: float64 [n_psd, 2, n_f]."""

    def __init__(self, resid, psd, k_lo, walker_psd=None, psd_is_inverse=False):
        assert resid.dtype == np.complex128 and resid.ndim == 3 and resid.shape[1] == 2
        assert resid.flags.c_contiguous
        self.resid = resid
        self.psd = np.ascontiguousarray(psd, dtype=np.float64)
        assert self.psd.ndim == 3 and self.psd.shape[1] == 2 and self.psd.shape[2] == resid.shape[2]
        self.walker_psd = None if walker_psd is None else np.ascontiguousarray(walker_psd, dtype=np.int32)
        self.k_lo = int(k_lo)
        self.psd_is_inverse = bool(psd_is_inverse)

    def c(self) -> _Data:
        return _Data(_ptr(self.resid), _ptr(self.psd), _ptr(self.walker_psd), self.k_lo,
                     self.resid.shape[2], self.resid.shape[0], self.psd.shape[0], int(self.psd_is_inverse))


def slow_envelope(cfg: Config, params, N: int):
    """A_s(t_n), E_s(t_n), n = 0..N-1 (steps O1-O5).  Returns two complex128 arrays [N]."""
    p = _f64(params)
    cc = cfg.c()
    a = np.empty(2, np.float64)
    e = np.empty(2, np.float64)
    As = np.empty(N, np.complex128)
    Es = np.empty(N, np.complex128)
    for n in range(N):
        lib().gbo_slow_envelope(C.byref(cc), _ptr(p), C.c_int(N), C.c_int(n), _ptr(a), _ptr(e))
        As[n] = a[0] + 1j * a[1]
        Es[n] = e[0] + 1j * e[1]
    return As, Es


def waveform(cfg: Config, params, N: int, use_dft: bool = False):
    """One source: returns (A[N], E[N], kmin) (steps O1-O6)."""
    p = _f64(params)
    A = np.empty(N, np.complex128)
    E = np.empty(N, np.complex128)
    kmin = C.c_int64(0)
    cc = cfg.c()
    rc = lib().gbo_waveform_ex(C.byref(cc), _ptr(p), C.c_int(N), C.c_int(int(use_dft)), _ptr(A), _ptr(E),
                               C.byref(kmin))
    if rc != 0:
        raise ValueError(f"gbo_waveform_ex rc={rc}")
    return A, E, int(kmin.value)


def waveform_batch(cfg: Config, params, N: int = 0, n_bins=None, nthreads: int = 1):
    """Batched: returns (AE[B,2,Nmax] complex128, kmin[B] int64); rows shorter than Nmax are zero padded."""
    p = _f64(params).reshape(-1, 8)
    B = p.shape[0]
    nb = None if n_bins is None else np.ascontiguousarray(n_bins, dtype=np.int32)
    Nmax = int(N if nb is None else (nb.max() if B else N))
    AE = np.zeros((B, 2, Nmax), np.complex128)
    kmin = np.zeros(B, np.int64)
    cc = cfg.c()
    rc = lib().gbo_waveform_batch(C.byref(cc), _ptr(p), C.c_int64(B), C.c_int(N), _ptr(nb), C.c_int(Nmax),
                                  _ptr(AE), _ptr(kmin), C.c_int(nthreads))
    if rc != 0:
        raise ValueError(f"gbo_waveform_batch rc={rc}")
    return AE, kmin


def delta_loglike(cfg: Config, data: Data, params_new, params_old, walker_index, move=None, move_all=ADD,
                  N: int = 0, n_bins=None, want_aux: bool = False, nthreads: int = 1):
    """Batched step O8.  Returns dlnL[B] (and aux[B,2] = (<h|h>, <r|h>) if want_aux)."""
    pn = None if params_new is None else _f64(params_new).reshape(-1, 8)
    po = None if params_old is None else _f64(params_old).reshape(-1, 8)
    w = np.ascontiguousarray(walker_index, dtype=np.int32)
    B = w.shape[0]
    mv = None if move is None else np.ascontiguousarray(move, dtype=np.int8)
    nb = None if n_bins is None else np.ascontiguousarray(n_bins, dtype=np.int32)
    out = np.zeros(B, np.float64)
    aux = np.zeros((B, 2), np.float64) if want_aux else None
    cc, dd = cfg.c(), data.c()
    rc = lib().gbo_delta_loglike(C.byref(cc), C.byref(dd), _ptr(pn), _ptr(po), _ptr(w), _ptr(mv),
                                 C.c_int(move_all), C.c_int(N), _ptr(nb), C.c_int64(B), _ptr(out), _ptr(aux),
                                 C.c_int(nthreads))
    if rc != 0:
        raise ValueError(f"gbo_delta_loglike rc={rc}")
    return (out, aux) if want_aux else out


def delta_loglike_accept(cfg: Config, data: Data, params_new, params_old, walker_index, logu, logq=None, beta=None,
                         move=None, move_all=ADD, N: int = 0, n_bins=None, apply: bool = True, nthreads: int = 1):
    """gbo_delta_loglike_accept: delta lnL of every row against one snapshot, accepted iff beta dlnL + logq >= logu, then
    (apply) the accepted rows update data.resid in place.  Returns (dlnL[B], accepted[B] uint8)."""
    pn = None if params_new is None else _f64(params_new).reshape(-1, 8)
    po = None if params_old is None else _f64(params_old).reshape(-1, 8)
    w = np.ascontiguousarray(walker_index, dtype=np.int32)
    B = w.shape[0]
    mv = None if move is None else np.ascontiguousarray(move, dtype=np.int8)
    nb = None if n_bins is None else np.ascontiguousarray(n_bins, dtype=np.int32)
    lu = _f64(logu)
    lq = None if logq is None else _f64(logq)
    bt = None if beta is None else _f64(beta)
    out, acc = np.zeros(B, np.float64), np.zeros(B, np.uint8)
    cc, dd = cfg.c(), data.c()
    rc = lib().gbo_delta_loglike_accept(C.byref(cc), C.byref(dd), _ptr(pn), _ptr(po), _ptr(w), _ptr(mv), C.c_int(move_all),
                                        C.c_int(N), _ptr(nb), C.c_int64(B), _ptr(lq), _ptr(lu), _ptr(bt), _ptr(out), None,
                                        _ptr(acc), C.c_int(1 if apply else 0), C.c_int(nthreads))
    if rc != 0:
        raise ValueError(f"gbo_delta_loglike_accept rc={rc}")
    return out, acc


def residual_update(cfg: Config, data: Data, params_new, params_old, walker_index, move=None, move_all=ADD,
                    accepted=None, N: int = 0, n_bins=None, nthreads: int = 1):
    """Step O9, in place on data.resid."""
    pn = None if params_new is None else _f64(params_new).reshape(-1, 8)
    po = None if params_old is None else _f64(params_old).reshape(-1, 8)
    w = np.ascontiguousarray(walker_index, dtype=np.int32)
    B = w.shape[0]
    mv = None if move is None else np.ascontiguousarray(move, dtype=np.int8)
    nb = None if n_bins is None else np.ascontiguousarray(n_bins, dtype=np.int32)
    acc = None if accepted is None else np.ascontiguousarray(accepted, dtype=np.uint8)
    cc, dd = cfg.c(), data.c()
    rc = lib().gbo_residual_update(C.byref(cc), C.byref(dd), _ptr(pn), _ptr(po), _ptr(w), _ptr(mv),
                                   C.c_int(move_all), _ptr(acc), C.c_int(N), _ptr(nb), C.c_int64(B),
                                   C.c_int(nthreads))
    if rc != 0:
        raise ValueError(f"gbo_residual_update rc={rc}")


def overlap(cfg: Config, data: Data, params_a, params_c, psd_row=None, N: int = 0, n_bins=None, nthreads: int = 1):
    """Normalised overlap <a|c>/sqrt(<a|a><c|c>) of B source pairs against PSD row psd_row[b] (row 0 if None).
    Returns (overlap[B], aux[B, 2] = (<a|a>, <c|c>)).  data.resid is not used."""
    pa, pc = _f64(params_a).reshape(-1, 8), _f64(params_c).reshape(-1, 8)
    B = pa.shape[0]
    pr = None if psd_row is None else np.ascontiguousarray(psd_row, dtype=np.int32)
    nb = None if n_bins is None else np.ascontiguousarray(n_bins, dtype=np.int32)
    out = np.zeros(B, np.float64)
    aux = np.zeros((B, 2), np.float64)
    cc, dd = cfg.c(), data.c()
    rc = lib().gbo_overlap(C.byref(cc), C.byref(dd), _ptr(pa), _ptr(pc), _ptr(pr), C.c_int(N), _ptr(nb), C.c_int64(B),
                           _ptr(out), _ptr(aux), C.c_int(nthreads))
    if rc != 0:
        raise ValueError(f"gbo_overlap rc={rc}")
    return out, aux


_BAND_TASK = np.dtype([("walker", np.int32), ("n_src", np.int32), ("src_begin", np.int32), ("n_prop", np.int32),
                       ("prop_begin", np.int32), ("n_stage", np.int32), ("k_first", np.int64),
                       ("flags", np.int32), ("write_walker", np.int32), ("beta", np.float64)], align=True)


def _pack_band_tasks(tasks: dict) -> np.ndarray:
    n = len(tasks["walker"])
    t = np.zeros(n, _BAND_TASK)
    for key in ("walker", "n_src", "src_begin", "n_prop", "prop_begin", "n_stage", "k_first", "beta"):
        t[key] = tasks[key]
    flags = (np.asarray(tasks["write_back"]) != 0).astype(np.int32)
    if "subtract_current" in tasks:
        flags |= 2 * (np.asarray(tasks["subtract_current"]) != 0).astype(np.int32)
    if "write_walker" in tasks:
        flags |= 4
        t["write_walker"] = tasks["write_walker"]
    t["flags"] = flags
    return t


def band_sweep(cfg: Config, data: Data, tasks: dict, N: int, params, prop_k, prop_params, prop_logq, prop_logu):
    """Algorithm 1, task after task, proposal after proposal.  `tasks` is a dict of equal-length
    arrays (walker, n_src, src_begin, n_prop, prop_begin, n_stage, k_first, write_back, beta; optional subtract_current
    and write_walker for the odd/even buffers of PAPER.md:354-362).  `params` [n_src_total, 8]
    and data.resid are updated in place.  Returns (accepted[n_prop_total] uint8, dlnL[n_prop_total])."""
    t = _pack_band_tasks(tasks)
    n = len(t)
    assert params.dtype == np.float64 and params.flags.c_contiguous
    pk = np.ascontiguousarray(prop_k, dtype=np.int32)
    pp, lq, lu = _f64(prop_params), _f64(prop_logq), _f64(prop_logu)
    acc = np.zeros(pk.shape[0], np.uint8)
    dl = np.zeros(pk.shape[0], np.float64)
    cc, dd = cfg.c(), data.c()
    rc = lib().gbo_band_sweep(C.byref(cc), C.byref(dd), _ptr(t), C.c_int64(n), C.c_int(N), _ptr(params), _ptr(pk),
                              _ptr(pp), _ptr(lq), _ptr(lu), _ptr(acc), _ptr(dl))
    if rc != 0:
        raise ValueError(f"gbo_band_sweep rc={rc}")
    return acc, dl


class _Stretch(C.Structure):
    _fields_ = [("seed", C.c_uint64), ("sweep", C.c_uint32), ("n_friends", C.c_int32), ("group", C.c_void_p),
                ("n_group", C.c_int64), ("stretch_a", C.c_double), ("lo", C.c_double * 8), ("hi", C.c_double * 8),
                ("periodic", C.c_int32 * 8)]


class Stretch:
    """Inputs of the in-loop proposal step of Algorithm 1 (gbo_stretch): Philox seed / sweep, the stationary group
    [n_group, 8] sorted by f0, n_friends, the stretch scale a, the prior box and the periodic flags."""

    def __init__(self, seed, sweep, group, n_friends, lo, hi, periodic, stretch_a=2.0):
        self.group = np.ascontiguousarray(group, dtype=np.float64)
        assert self.group.ndim == 2 and self.group.shape[1] == 8
        assert np.all(np.diff(self.group[:, 1]) >= 0), "the stationary group must be sorted by f0"
        self.seed, self.sweep, self.n_friends, self.stretch_a = int(seed), int(sweep), int(n_friends), float(stretch_a)
        self.lo, self.hi = np.asarray(lo, np.float64), np.asarray(hi, np.float64)
        self.periodic = np.asarray(periodic, np.int32)

    def c(self) -> _Stretch:
        return _Stretch(self.seed, self.sweep, self.n_friends, _ptr(self.group), self.group.shape[0], self.stretch_a,
                        (C.c_double * 8)(*self.lo), (C.c_double * 8)(*self.hi), (C.c_int32 * 8)(*self.periodic))


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(x) for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) for x in key])
    out = (C.c_uint32 * 4)()
    lib().gbo_philox4x32_10(c, k, out)
    return [int(x) for x in out]


def uniform52(w0: int, w1: int) -> float:
    f = lib().gbo_uniform52
    f.restype = C.c_double
    return float(f(C.c_uint32(w0), C.c_uint32(w1)))


def randint(w: int, n: int) -> int:
    return int(lib().gbo_randint(C.c_uint32(w), C.c_int32(n)))


def stretch_z(u: float, a: float = 2.0) -> float:
    f = lib().gbo_stretch_z
    f.restype = C.c_double
    return float(f(C.c_double(u), C.c_double(a)))


def friend_row(group, n_friends: int, f: float, j: int) -> int:
    g = np.ascontiguousarray(group, dtype=np.float64)
    fn = lib().gbo_friend_row
    fn.restype = C.c_int64
    return int(fn(_ptr(g), C.c_int64(g.shape[0]), C.c_int32(n_friends), C.c_double(f), C.c_int32(j)))


def make_proposal(st: Stretch, row: int, theta):
    """One proposal for global proposal row `row` of a band whose current sources are theta [g_j, 8].
    Returns (inside_prior, k, theta' [8], logq, logu)."""
    th = np.ascontiguousarray(theta, dtype=np.float64)
    k = C.c_int32(0)
    out = np.empty(8)
    lq, lu = C.c_double(0.0), C.c_double(0.0)
    sc = st.c()
    inside = lib().gbo_make_proposal(C.byref(sc), C.c_int64(row), _ptr(th), C.c_int32(th.shape[0]), C.byref(k), _ptr(out),
                                     C.byref(lq), C.byref(lu))
    return bool(inside), int(k.value), out, float(lq.value), float(lu.value)


def band_sweep_generate(cfg: Config, data: Data, tasks: dict, N: int, params, st: Stretch):
    """Algorithm 1 with the proposal step inside the loop (gbo_band_sweep_generate).  `params` and data.resid are updated
    in place.  Returns (accepted uint8, dlnL, k int32, theta' [P, 8], logq, logu) over all proposal rows."""
    t = _pack_band_tasks(tasks)
    assert params.dtype == np.float64 and params.flags.c_contiguous
    P = int((t["prop_begin"] + t["n_prop"]).max()) if len(t) else 0
    acc, dl = np.zeros(P, np.uint8), np.zeros(P)
    k, pp, lq, lu = np.zeros(P, np.int32), np.zeros((P, 8)), np.zeros(P), np.zeros(P)
    cc, dd, sc = cfg.c(), data.c(), st.c()
    rc = lib().gbo_band_sweep_generate(C.byref(cc), C.byref(dd), _ptr(t), C.c_int64(len(t)), C.c_int(N), _ptr(params),
                                       C.byref(sc), _ptr(k), _ptr(pp), _ptr(lq), _ptr(lu), _ptr(acc), _ptr(dl))
    if rc != 0:
        raise ValueError(f"gbo_band_sweep_generate rc={rc}")
    return acc, dl, k, pp, lq, lu


_TEMPER_TASK = np.dtype([("n_t", np.int32), ("chain_begin", np.int32), ("n_stage", np.int32), ("write_back", np.int32),
                         ("k_first", np.int64), ("write_walker", np.int32), ("reserved", np.int32)], align=True)


def temper_sweep(cfg: Config, data: Data, tasks: dict, N: int, params, chain_walker, chain_beta, chain_set_begin,
                 chain_set_n, chain_logu):
    """Algorithm 2 with Eq. D2, task after task.  `tasks`: dict of equal-length arrays n_t, chain_begin,
    n_stage, write_back, k_first; an optional write_walker column selects the odd/even cold-chain buffer mode (every
    chain's residual is formed as its walker's row minus the set it holds; only exchanges with the cold chain are written,
    into row write_walker).  data.resid is updated in place.
    Returns (perm[n_chain] int32, accepted[n_chain] uint8, dlnl[n_chain, 2])."""
    n = len(tasks["n_t"])
    t = np.zeros(n, _TEMPER_TASK)
    for key in ("n_t", "chain_begin", "n_stage", "write_back", "k_first"):
        t[key] = tasks[key]
    if "write_walker" in tasks:          # odd/even cold-chain buffers: bit 2 of write_back + the cold row
        t["write_back"] = (np.asarray(tasks["write_back"]) != 0).astype(np.int32) | 2
        t["write_walker"] = tasks["write_walker"]
    p = _f64(params)
    cw = np.ascontiguousarray(chain_walker, dtype=np.int32)
    sb = np.ascontiguousarray(chain_set_begin, dtype=np.int32)
    sn = np.ascontiguousarray(chain_set_n, dtype=np.int32)
    cb, lu = _f64(chain_beta), _f64(chain_logu)
    nc = cw.shape[0]
    perm = np.zeros(nc, np.int32)
    acc = np.zeros(nc, np.uint8)
    dl = np.zeros((nc, 2), np.float64)
    cc, dd = cfg.c(), data.c()
    rc = lib().gbo_temper_sweep(C.byref(cc), C.byref(dd), _ptr(t), C.c_int64(n), C.c_int(N), _ptr(p), _ptr(cw), _ptr(cb),
                                _ptr(sb), _ptr(sn), _ptr(lu), _ptr(perm), _ptr(acc), _ptr(dl))
    if rc != 0:
        raise ValueError(f"gbo_temper_sweep rc={rc}")
    return perm, acc, dl


def inner_windows(cfg: Config, data: Data, psd_row: int, bA, bE, kb: int, cA, cE, kc: int) -> float:
    """<b|c> of two explicit windows (step O7)."""
    bA, bE, cA, cE = (np.ascontiguousarray(z, dtype=np.complex128) for z in (bA, bE, cA, cE))
    cc, dd = cfg.c(), data.c()
    return float(lib().gbo_inner_windows(C.byref(cc), C.byref(dd), C.c_int(psd_row),
                                         _ptr(bA), _ptr(bE), C.c_int64(kb), C.c_int(len(bA)),
                                         _ptr(cA), _ptr(cE), C.c_int64(kc), C.c_int(len(cA))))


def dft(x):
    x = np.ascontiguousarray(x, dtype=np.complex128)
    F = np.empty_like(x)
    lib().gbo_dft(_ptr(x), C.c_int(len(x)), _ptr(F))
    return F


def fft(x):
    x = np.ascontiguousarray(x, dtype=np.complex128)
    F = np.empty_like(x)
    rc = lib().gbo_fft(_ptr(x), C.c_int(len(x)), _ptr(F))
    if rc != 0:
        raise ValueError("gbo_fft: N must be a power of two")
    return F


def orbits(cfg: Config, t: float):
    x = np.empty((3, 3), np.float64)
    cc = cfg.c()
    lib().gbo_orbits(C.byref(cc), C.c_double(t), _ptr(x))
    return x
