"""Host logic of the product path's arithmetic (no GPU): tests/host_replay.cpp replays, on the CPU, the per-sample
functions and FFT stages the CUDA kernels run, and this file compares them with the oracle.

This pins the restructured slow part of csrc/gb_fast.cuh (polynomial sin/cos, multiple-angle phasors, shared
reciprocal) and the general path of csrc/gb_math.cuh against the oracle at the north_star tolerance
(1e-9 of the peak bin; the observed level is ~1e-13) before any GPU time is spent.  The GPU parity tests
(-m gpu) remain the parity tests proper.
"""
import ctypes as C
import os
import subprocess
import tempfile

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "tests", "host_replay.cpp")


@pytest.fixture(scope="module")
def replay():
    out = os.path.join(tempfile.mkdtemp(prefix="gb_replay_"), "libgb_replay.so")
    cmd = ["g++", "-std=c++17", "-O2", "-mfma", "-ffp-contract=off", "-shared", "-fPIC", "-x", "c++", SRC, "-o", out]
    subprocess.run(cmd, check=True)
    lib = C.CDLL(out)
    lib.gb_replay_waveform.restype = C.c_int
    lib.gb_replay_fast_ok.restype = C.c_int
    return lib


def _wave(lib, cfg, p, N, path):
    p = np.ascontiguousarray(p, np.float64)
    AE = np.empty((2, N), np.complex128)
    kmin = C.c_int64(0)
    used = C.c_int(0)
    rc = lib.gb_replay_waveform(p.ctypes.data_as(C.c_void_p), C.c_int(N), C.c_double(cfg.Tobs),
                                C.c_double(cfg.armlength), C.c_double(cfg.au), C.c_double(cfg.year),
                                C.c_double(cfg.kappa), C.c_double(cfg.lambda0), C.c_int(path),
                                AE.ctypes.data_as(C.c_void_p), C.byref(kmin), C.byref(used))
    assert rc == 0
    return AE, int(kmin.value), int(used.value)


def _params(seed, B, f_lo, f_hi, fdot=1e-16):
    g = np.random.default_rng(seed)
    u = g.random((B, 8))
    p = np.empty((B, 8))
    p[:, 0] = 10.0 ** (-23 + 2 * u[:, 0])
    p[:, 1] = f_lo * (f_hi / f_lo) ** u[:, 1]
    p[:, 2] = (2 * u[:, 2] - 1) * fdot
    p[:, 3] = 2 * np.pi * u[:, 3]
    p[:, 4] = 2 * u[:, 4] - 1
    p[:, 5] = np.pi * u[:, 5]
    p[:, 6] = 2 * np.pi * u[:, 6]
    p[:, 7] = 2 * u[:, 7] - 1
    return p


def _err(AE, ref):
    return float(np.abs(AE - ref).max() / np.abs(ref).max())


@pytest.mark.parametrize("N,f_lo,f_hi", [(128, 1e-4, 1e-3), (256, 1e-3, 4e-3), (512, 4e-3, 1e-2), (1024, 1e-2, 3e-2)])
def test_fast_and_general_paths_match_oracle(oracle, replay, N, f_lo, f_hi):
    cfg = oracle.Config()
    worst = {0: 0.0, 1: 0.0}
    for p in _params(100 + N, 24, f_lo, f_hi):
        A, E, kmin = oracle.waveform(cfg, p, N)
        ref = np.stack([A, E])
        for path in (0, 1):
            AE, k, used = _wave(replay, cfg, p, N, path)
            assert k == kmin and used == path
            worst[path] = max(worst[path], _err(AE, ref))
    assert worst[0] < 1e-11 and worst[1] < 1e-11, worst


def test_fast_path_with_large_fdot_and_any_window_length(oracle, replay):
    """fdot up to 1e-13 Hz/s (eps_r ~ 2e-9 rad, first order) and window lengths not tied to f0."""
    cfg = oracle.Config()
    worst = 0.0
    for i, p in enumerate(_params(7, 16, 2e-4, 2.9e-2, fdot=1e-13)):
        N = (128, 256, 512, 1024)[i % 4]
        assert replay.gb_replay_fast_ok(p.ctypes.data_as(C.c_void_p), C.c_double(cfg.Tobs), C.c_double(cfg.armlength),
                                        C.c_double(cfg.au)) == 1
        A, E, kmin = oracle.waveform(cfg, p, N)
        AE, k, used = _wave(replay, cfg, p, N, 2)
        assert used == 1 and k == kmin
        worst = max(worst, _err(AE, np.stack([A, E])))
    assert worst < 1e-10, worst


def test_rows_outside_the_fast_limits_take_the_general_path(oracle, replay):
    cfg = oracle.Config()
    base = _params(3, 1, 2e-3, 3e-3)[0]
    cases = []
    for k, v in ((1, 4.5e-2), (2, 5e-12), (3, 4000.0), (1, -1e-3), (1, float("nan"))):
        p = base.copy()
        p[k] = v
        cases.append(p)
    for p in cases:
        ok = replay.gb_replay_fast_ok(p.ctypes.data_as(C.c_void_p), C.c_double(cfg.Tobs), C.c_double(cfg.armlength),
                                      C.c_double(cfg.au))
        assert ok == 0
    # a 45 mHz source (beyond the fast limit, below Nyquist) through the dispatcher: general path, still exact
    p = cases[0]
    A, E, kmin = oracle.waveform(cfg, p, 1024)
    AE, k, used = _wave(replay, cfg, p, 1024, 2)
    assert used == 0 and k == kmin and _err(AE, np.stack([A, E])) < 1e-11


def test_source_along_a_link_direction_takes_the_series_branch(oracle, replay):
    """kappa -> +-1 at some samples: the shared reciprocal is singular there, the sinc series takes over."""
    cfg = oracle.Config()
    # link vectors at t = 0 from the oracle's orbits; aim the propagation direction k along n_12 and n_31
    x = oracle.orbits(cfg, 0.0)
    worst = 0.0
    for (r, s_), sign in (((0, 1), 1.0), ((2, 0), -1.0), ((1, 2), 1.0)):
        n = (x[r] - x[s_]) / cfg.armlength
        n /= np.linalg.norm(n)
        kdir = sign * n                      # k = -(cos b cos l, cos b sin l, sin b)
        sinb = -kdir[2]
        lam = np.arctan2(-kdir[1], -kdir[0]) % (2 * np.pi)
        for f0 in (3e-4, 6e-3):
            p = np.array([1e-22, f0, 1e-17, 1.0, 0.3, 0.7, lam, sinb])
            N = 256
            A, E, kmin = oracle.waveform(cfg, p, N)
            AE, k, used = _wave(replay, cfg, p, N, 1)
            worst = max(worst, _err(AE, np.stack([A, E])))
    assert worst < 1e-10, worst


def test_bounded_range_sincos_accuracy(replay):
    g = np.random.default_rng(11)
    for which, R in ((0, 0.8), (1, 0.27), (2, 2999.0)):
        x = np.concatenate([g.uniform(-R, R, 20000), [0.0, R, -R, 1e-300, 1e-9, -1e-9]])
        s = np.empty_like(x)
        c = np.empty_like(x)
        replay.gb_replay_sincos(C.c_int(which), x.ctypes.data_as(C.c_void_p), C.c_int(x.size),
                                s.ctypes.data_as(C.c_void_p), c.ctypes.data_as(C.c_void_p))
        xl = x.astype(np.longdouble)
        es = np.abs(s - np.sin(xl)).astype(np.float64)
        ec = np.abs(c - np.cos(xl)).astype(np.float64)
        if which < 2:   # relative accuracy of the sine is kept down to x -> 0
            rel = es[x != 0] / np.abs(np.sin(xl[x != 0])).astype(np.float64)
            assert rel.max() < 4e-16, (which, rel.max())
        assert es.max() < 4e-16 and ec.max() < 4e-16, (which, es.max(), ec.max())
