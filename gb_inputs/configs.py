"""Workload recipes for BASELINE.json configs 1..5.

Random numbers: numpy's counter-based Philox4x64 (np.random.Philox(key=...)), keyed by
(SEED_BASE + config index, stream id); uniforms are numpy's 53-bit doubles, normals numpy's ziggurat.
Every array is a pure function of (config index, sizes), so oracle and GPU always see the same inputs.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

TOBS = 31457280.0          # 1 "year" of the configs = 3 * 2^21 * 5 s
DT = 5.0
C_LIGHT = 299792458.0
ARMLENGTH = 2.5e9
SEED_BASE = 0x2405_0469_0000
ADD, REMOVE, SWAP = 0, 1, 2

# stream ids within one config's key space
_S_PARAMS, _S_WALKER, _S_MOVE, _S_JITTER, _S_ACCEPT, _S_PSD, _S_NOISE0 = 1, 2, 3, 4, 5, 6, 1000


def _rng(config: int, stream: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[SEED_BASE + config, stream]))


def band_bins(f_lo: float, f_hi: float, T: float = TOBS):
    """Global rfft bin range [k_lo, k_lo + n_f) covering f_lo..f_hi inclusive (bin k <-> f = k/T)."""
    k_lo = int(np.ceil(f_lo * T - 1e-9))
    k_hi = int(np.floor(f_hi * T + 1e-9))
    return k_lo, k_hi - k_lo + 1


def n_bins_for_f0(f0):
    """Window length by f0 (BASELINE.json config 3/5): 128 (<1 mHz), 256 (1-4), 512 (4-10), 1024 above."""
    f0 = np.asarray(f0)
    return np.where(f0 < 1e-3, 128, np.where(f0 < 4e-3, 256, np.where(f0 < 10e-3, 512, 1024))).astype(np.int32)


def instrument_psd(f, sqrt_S_acc: float = 3e-15, sqrt_S_oms: float = 15e-12, L: float = ARMLENGTH):
    """A/E instrument noise PSD, Eq. 7-9, fractional-frequency TDI-1.5 units [1/Hz]."""
    f = np.asarray(f, dtype=np.float64)
    x = 2.0 * np.pi * f * L / C_LIGHT
    S_pm = sqrt_S_acc ** 2 * (2.0 * np.pi * C_LIGHT * f) ** -2 * (1.0 + (0.4e-3 / f) ** 2) * (1.0 + (f / 8e-3) ** 4)
    S_op = sqrt_S_oms ** 2 * (2.0 * np.pi * f / C_LIGHT) ** 2 * (1.0 + (2e-3 / f) ** 4)
    return 8.0 * np.sin(x) ** 2 * (2.0 * S_pm * (3.0 + 2.0 * np.cos(x) + np.cos(2.0 * x)) + S_op * (2.0 + np.cos(x)))


def _draw_params(g: np.random.Generator, B: int, f_lo: float, f_hi: float):
    """[amp, f0, fdot, phi0, cos_iota, psi, lambda, sin_beta] per BASELINE.json config 1."""
    p = np.empty((B, 8), np.float64)
    u = g.random((B, 8))
    p[:, 0] = 10.0 ** (-23.0 + 2.0 * u[:, 0])                       # amp log-U[1e-23, 1e-21]
    p[:, 1] = f_lo * (f_hi / f_lo) ** u[:, 1]                       # f0 log-U
    p[:, 2] = (2.0 * u[:, 2] - 1.0) * 1e-16                         # fdot U[-1e-16, 1e-16]
    p[:, 3] = 2.0 * np.pi * u[:, 3]                                 # phi0
    p[:, 4] = 2.0 * u[:, 4] - 1.0                                   # cos iota
    p[:, 5] = np.pi * u[:, 5]                                       # psi
    p[:, 6] = 2.0 * np.pi * u[:, 6]                                 # lambda
    p[:, 7] = 2.0 * u[:, 7] - 1.0                                   # sin beta
    return p


# calibration constant of the config-5 amplitude recipe: rho0^2 = T (amp0 * _RESP_C0 * x |sin x|)^2 / S(f0)
# approximates the orientation-averaged optimal SNR of a source of amplitude amp0 (value immaterial to parity)
_RESP_C0 = 4.74


@dataclass
class Workload:
    config: int
    name: str
    Tobs: float
    dt: float
    k_lo: int
    n_f: int
    n_walkers: int
    psd: np.ndarray                      # [n_psd, 2, n_f] f64, S_n
    walker_psd: Optional[np.ndarray]     # [n_walkers] int32 or None
    params_new: Optional[np.ndarray]     # [B, 8]
    params_old: Optional[np.ndarray]     # [B, 8]
    walker_index: np.ndarray             # [B] int32
    move: Optional[np.ndarray]           # [B] int8 or None
    move_all: int
    N: int                               # used when n_bins is None
    n_bins: Optional[np.ndarray]         # [B] int32 or None
    accepted: Optional[np.ndarray]       # [B] uint8 or None
    _psd_scale: np.ndarray = field(default=None, repr=False)

    @property
    def B(self) -> int:
        return int(self.walker_index.shape[0])

    def psd_row_of(self, w: int) -> int:
        if self.walker_psd is not None:
            return int(self.walker_psd[w])
        return 0 if self.psd.shape[0] == 1 else w

    def resid_row(self, w: int) -> np.ndarray:
        """Residual of walker w: complex128 [2, n_f], Re and Im ~ N(0, S T / 4) (P7 normalisation)."""
        g = _rng(self.config, _S_NOISE0 + w)
        z = g.standard_normal((2, self.n_f, 2))
        sig = np.sqrt(self.psd[self.psd_row_of(w)] * (self.Tobs / 4.0))
        out = np.empty((2, self.n_f), np.complex128)
        out.real = z[..., 0] * sig
        out.imag = z[..., 1] * sig
        return out

    def resid(self) -> np.ndarray:
        """All residuals: complex128 [n_walkers, 2, n_f] (config 5 full size: 10.8 GB -- use resid_row)."""
        out = np.empty((self.n_walkers, 2, self.n_f), np.complex128)
        for w in range(self.n_walkers):
            out[w] = self.resid_row(w)
        return out

    def subset(self, idx) -> "Workload":
        """Same data, a subset of the proposal rows (for sampled parity / bounded CPU baselines)."""
        idx = np.asarray(idx)
        pick = lambda a: None if a is None else np.ascontiguousarray(a[idx])
        return Workload(self.config, self.name, self.Tobs, self.dt, self.k_lo, self.n_f, self.n_walkers,
                        self.psd, self.walker_psd, pick(self.params_new), pick(self.params_old),
                        pick(self.walker_index), pick(self.move), self.move_all, self.N, pick(self.n_bins),
                        pick(self.accepted), self._psd_scale)


# E-channel noise levels of the un-jittered configs 1-2 relative to the A channel.  The paper fits the noise
# "in both channels (i.e., four parameters in total)", so S_A != S_E is the normal case; a fixed
# offset keeps every PSD row's two channels distinguishable, so that a swapped or duplicated channel row cannot
# pass a parity test.
_E_OFFSET = (1.04, 0.97)      # (sqrt S_acc, sqrt S_oms) of E / nominal


def _psd_rows(config: int, n_rows: int, k_lo: int, n_f: int, jitter: bool):
    """PSD rows [n_rows, 2, n_f]: channel 0 = A, channel 1 = E, each with its own (sqrt S_acc, sqrt S_oms) pair
    (four noise parameters, two per channel).  Returns (psd, scale[n_rows, 2 channels, 2 levels])."""
    f = (k_lo + np.arange(n_f, dtype=np.float64)) / TOBS
    psd = np.empty((n_rows, 2, n_f), np.float64)
    g = _rng(config, _S_PSD)
    scale = np.ones((n_rows, 2, 2))
    if jitter:
        scale[:, 0, :] = 1.0 + 0.05 * (2.0 * g.random((n_rows, 2)) - 1.0)      # A: the draws of the first recipe
        scale[:, 1, :] = 1.0 + 0.05 * (2.0 * g.random((n_rows, 2)) - 1.0)      # E: its own draws
    else:
        scale[:, 1, :] = _E_OFFSET
    for r in range(n_rows):
        for ch in range(2):
            psd[r, ch] = instrument_psd(f, 3e-15 * scale[r, ch, 0], 15e-12 * scale[r, ch, 1])
    return psd, scale


def make_workload(config: int, B: Optional[int] = None, n_walkers: Optional[int] = None,
                  per_walker: Optional[int] = None) -> Workload:
    """Build config 1..5.  B / n_walkers / per_walker shrink the case for tests; the draws for a
    smaller B are a prefix of the draws for a larger one (same Philox streams)."""
    if config == 1:
        B = 64 if B is None else B
        k_lo, n_f = band_bins(1e-3, 4e-3)
        psd, sc = _psd_rows(1, 1, k_lo, n_f, False)
        p = _draw_params(_rng(1, _S_PARAMS), B, 1e-3, 4e-3)
        return Workload(1, "cfg1_tiny_add", TOBS, DT, k_lo, n_f, 1, psd, None, p, None,
                        np.zeros(B, np.int32), None, ADD, 128, None, None, sc)
    if config == 2:
        B = 4096 if B is None else B
        k_lo, n_f = band_bins(0.1e-3, 30e-3)
        psd, sc = _psd_rows(2, 1, k_lo, n_f, False)
        p = _draw_params(_rng(2, _S_PARAMS), B, 0.1e-3, 15e-3)
        return Workload(2, "cfg2_add4096", TOBS, DT, k_lo, n_f, 1, psd, None, p, None,
                        np.zeros(B, np.int32), None, ADD, 256, None, None, sc)
    if config == 3:
        B = 65536 if B is None else B
        nw = 36 if n_walkers is None else n_walkers
        k_lo, n_f = band_bins(0.1e-3, 30e-3)
        psd, sc = _psd_rows(3, nw, k_lo, n_f, True)
        p = _draw_params(_rng(3, _S_PARAMS), B, 0.1e-3, 15e-3)
        w = _rng(3, _S_WALKER).integers(0, nw, B).astype(np.int32)
        mv = (_rng(3, _S_MOVE).random(B) < 0.5).astype(np.int8)      # 0 = ADD, 1 = REMOVE
        # ADD rows read params_new, REMOVE rows read params_old: hand the same draw to both
        return Workload(3, "cfg3_mixed_add_remove", TOBS, DT, k_lo, n_f, nw, psd, None, p, p.copy(),
                        w, mv, ADD, 0, n_bins_for_f0(p[:, 1]), None, sc)
    if config == 4:
        B = 32768 if B is None else B
        nw = 36 if n_walkers is None else n_walkers
        k_lo, n_f = band_bins(0.1e-3, 30e-3)
        psd, sc = _psd_rows(4, nw, k_lo, n_f, True)
        old = _draw_params(_rng(4, _S_PARAMS), B, 4e-3, 10e-3)
        g = _rng(4, _S_JITTER).standard_normal((B, 8))
        new = old.copy()
        new[:, 0] = old[:, 0] * (1.0 + 0.01 * g[:, 0])
        new[:, 1] = old[:, 1] + 1e-9 * g[:, 1]
        new[:, 3] = old[:, 3] + 0.05 * g[:, 3]
        new[:, 5] = old[:, 5] + 0.05 * g[:, 5]
        new[:, 6] = old[:, 6] + 0.05 * g[:, 6]
        iota = np.arccos(old[:, 4]) + 0.05 * g[:, 4]                 # reflect into [0, pi]
        iota = np.abs(iota); iota = np.where(iota > np.pi, 2.0 * np.pi - iota, iota)
        new[:, 4] = np.cos(iota)
        beta = np.arcsin(old[:, 7]) + 0.05 * g[:, 7]                 # reflect into [-pi/2, pi/2]
        beta = np.where(beta > np.pi / 2, np.pi - beta, beta); beta = np.where(beta < -np.pi / 2, -np.pi - beta, beta)
        new[:, 7] = np.sin(beta)
        w = _rng(4, _S_WALKER).integers(0, nw, B).astype(np.int32)
        return Workload(4, "cfg4_swap", TOBS, DT, k_lo, n_f, nw, psd, None, new, old,
                        w, None, SWAP, 512, None, None, sc)
    if config == 5:
        n_t, n_w36 = 10, 36
        nw = n_t * n_w36 if n_walkers is None else n_walkers
        per = 12000 if per_walker is None else per_walker
        B = nw * per if B is None else B
        k_lo, n_f = band_bins(0.1e-3, 30e-3)
        n_rows = min(n_w36, nw)
        psd, sc = _psd_rows(5, n_rows, k_lo, n_f, True)
        walker_psd = (np.arange(nw) % n_rows).astype(np.int32)       # "vertical" PSD sharing across temps
        p = _draw_params(_rng(5, _S_PARAMS), B, 0.1e-3, 15e-3)
        # SNR-weighted amplitude: rho ~ p(rho) ∝ rho^-4 on [7, 500] (inverse CDF), amp = amp0 rho / rho0(f0)
        u = p[:, 0].copy(); u = (np.log10(u) + 23.0) / 2.0            # recover the uniform behind column 0
        lo, hi = 7.0, 500.0
        rho = (lo ** -3 - u * (lo ** -3 - hi ** -3)) ** (-1.0 / 3.0)
        f0 = p[:, 1]
        x = 2.0 * np.pi * f0 * ARMLENGTH / C_LIGHT
        amp0 = 1e-22
        rho0 = np.sqrt(TOBS / instrument_psd(f0)) * amp0 * _RESP_C0 * x * np.abs(np.sin(x))
        p[:, 0] = amp0 * rho / rho0
        w = (np.arange(B) // per).astype(np.int32) if B == nw * per else \
            _rng(5, _S_WALKER).integers(0, nw, B).astype(np.int32)
        acc = (_rng(5, _S_ACCEPT).random(B) < 0.25).astype(np.uint8)
        return Workload(5, "cfg5_ensemble_sweep", TOBS, DT, k_lo, n_f, nw, psd, walker_psd, p, None,
                        w, None, ADD, 0, n_bins_for_f0(p[:, 1]), acc, sc)
    raise ValueError(f"unknown config {config}")


# ---------------------------------------------------------------------------------------------------------
# Band tasks for the Algorithm-1 primitive: sub-bands of N bins
# (PAPER.md:288), one task per (walker, ODD sub-band) -- the paper's odd/even schedule -- staging
# sub-bands b-1, b, b+1; n_src sources with f0 inside sub-band b; n_prop proposals "theta' = theta + jitter" on
# randomly picked sources of the band (PAPER.md:595 randint), each with its log-uniform draw.
_S_BAND = 7


@dataclass
class BandTasks:
    N: int
    tasks: dict                 # equal-length arrays: walker, n_src, src_begin, n_prop, prop_begin, n_stage, k_first,
                                # write_back, beta
    params: np.ndarray          # [n_src_total, 8] current sources (in/out)
    prop_k: np.ndarray          # [n_prop_total] int32 index of the source within its band
    prop_params: np.ndarray     # [n_prop_total, 8]
    prop_logq: np.ndarray       # [n_prop_total] log prior/proposal ratio term (0 here)
    prop_logu: np.ndarray       # [n_prop_total] log of the uniform draw
    max_stage: int


def make_band_tasks(wl: Workload, N: int, f_lo: float, n_bands: int, n_src: int, n_prop: int,
                    betas=(1.0, 0.6), stream: int = 0, amp_lo: float = 2e-23, amp_hi: float = 2e-22,
                    band_stride: int = 2) -> BandTasks:
    """n_bands odd sub-bands per walker of `wl`, starting near f_lo.  Deterministic in (wl.config, N, stream).
    band_stride = 2: every odd sub-band (the paper's schedule; bands b and b + 2 both stage sub-band b + 1);
    band_stride = 4: every other odd sub-band, so the staged ranges of one walker's tasks are disjoint and the result of
    a sweep does not depend on the order in which the tasks run even when proposals roam over the whole stage."""
    g = _rng(wl.config, 100 * _S_BAND + stream + N)
    T = wl.Tobs
    kb0 = int(np.ceil(f_lo * T / N)) * N                       # global bin of sub-band 0 (a multiple of N)
    nw = wl.n_walkers
    nt = nw * n_bands
    walker = np.repeat(np.arange(nw, dtype=np.int32), n_bands)
    b = np.tile(band_stride * np.arange(n_bands, dtype=np.int64) + 1, nw)  # odd sub-bands
    tasks = {
        "walker": walker,
        "n_src": np.full(nt, n_src, np.int32),
        "src_begin": (np.arange(nt) * n_src).astype(np.int32),
        "n_prop": np.full(nt, n_prop, np.int32),
        "prop_begin": (np.arange(nt) * n_prop).astype(np.int32),
        "n_stage": np.full(nt, 3 * N, np.int32),
        "k_first": kb0 + (b - 1) * N,
        "write_back": np.ones(nt, np.int32),
        "beta": np.asarray(betas, np.float64)[walker % len(betas)],
    }
    u = g.random((nt, n_src, 8))
    p = np.empty((nt, n_src, 8))
    p[..., 0] = amp_lo * (amp_hi / amp_lo) ** u[..., 0]
    p[..., 1] = (kb0 + (b[:, None] + u[..., 1]) * N) / T          # f0 inside sub-band b
    p[..., 2] = (2.0 * u[..., 2] - 1.0) * 1e-16
    p[..., 3] = 2.0 * np.pi * u[..., 3]
    p[..., 4] = 2.0 * u[..., 4] - 1.0
    p[..., 5] = np.pi * u[..., 5]
    p[..., 6] = 2.0 * np.pi * u[..., 6]
    p[..., 7] = 2.0 * u[..., 7] - 1.0
    params = np.ascontiguousarray(p.reshape(nt * n_src, 8))
    prop_k = g.integers(0, n_src, (nt, n_prop)).astype(np.int32)
    z = g.standard_normal((nt, n_prop, 8))
    base = p[np.arange(nt)[:, None], prop_k]                     # proposals jitter the INITIAL parameters
    q = base.copy()
    q[..., 0] = base[..., 0] * (1.0 + 0.02 * z[..., 0])
    q[..., 1] = base[..., 1] + 2e-9 * z[..., 1]
    q[..., 3] = base[..., 3] + 0.05 * z[..., 3]
    q[..., 5] = base[..., 5] + 0.05 * z[..., 5]
    q[..., 6] = base[..., 6] + 0.02 * z[..., 6]
    q[..., 4] = np.clip(base[..., 4] + 0.02 * z[..., 4], -1.0, 1.0)
    q[..., 7] = np.clip(base[..., 7] + 0.02 * z[..., 7], -1.0, 1.0)
    logu = np.log(g.random((nt, n_prop)))
    return BandTasks(N, tasks, params, np.ascontiguousarray(prop_k.reshape(-1)),
                     np.ascontiguousarray(q.reshape(nt * n_prop, 8)), np.zeros(nt * n_prop),
                     np.ascontiguousarray(logu.reshape(-1)), 3 * N)


# ---------------------------------------------------------------------------------------------------------
# Inputs of the in-loop proposal step of Algorithm 1 (group stretch, App. B :566-576): the stationary
# group -- "a flattened set of all templates contained in the cold-chain in all current walkers", sorted by frequency
# -- stands in as n_copies jittered copies of every band's initial sources (what posterior samples of the
# same sources in other walkers look like), plus the prior box and the periodic flags of the 8 coordinates.
@dataclass
class StretchInputs:
    seed: int
    sweep: int
    group: np.ndarray           # [n_group, 8] sorted by f0 ascending
    n_friends: int
    stretch_a: float
    lo: np.ndarray              # [8] prior box
    hi: np.ndarray
    periodic: np.ndarray        # [8] int32


PRIOR_LO = np.array([1e-24, 5e-5, -1e-14, 0.0, -1.0, 0.0, 0.0, -1.0])
PRIOR_HI = np.array([1e-20, 3.1e-2, 1e-14, 2.0 * np.pi, 1.0, np.pi, 2.0 * np.pi, 1.0])
PERIODIC = np.array([0, 0, 0, 1, 0, 1, 1, 0], np.int32)      # phi0, psi, lambda


def make_stretch_inputs(bt: BandTasks, config: int = 3, n_copies: int = 12, n_friends: int = 24, seed: int = 0x2405,
                        sweep: int = 1, scale: float = 1.0) -> StretchInputs:
    g = _rng(config, 300 * _S_BAND + bt.N)
    base = np.repeat(bt.params, n_copies, axis=0)
    z = g.standard_normal(base.shape) * scale
    grp = base.copy()
    grp[:, 0] = base[:, 0] * (1.0 + 0.02 * z[:, 0])
    grp[:, 1] = base[:, 1] + 2e-9 * z[:, 1]
    grp[:, 2] = base[:, 2] + 2e-17 * z[:, 2]
    grp[:, 3] = np.mod(base[:, 3] + 0.05 * z[:, 3], 2.0 * np.pi)
    grp[:, 4] = np.clip(base[:, 4] + 0.02 * z[:, 4], -1.0, 1.0)
    grp[:, 5] = np.mod(base[:, 5] + 0.05 * z[:, 5], np.pi)
    grp[:, 6] = np.mod(base[:, 6] + 0.02 * z[:, 6], 2.0 * np.pi)
    grp[:, 7] = np.clip(base[:, 7] + 0.02 * z[:, 7], -1.0, 1.0)
    grp = np.ascontiguousarray(grp[np.argsort(grp[:, 1], kind="stable")])
    return StretchInputs(seed, sweep, grp, n_friends, 2.0, PRIOR_LO.copy(), PRIOR_HI.copy(), PERIODIC.copy())


# ---------------------------------------------------------------------------------------------------------
# Temperature-swap tasks for the Algorithm-2 primitive: one task per
# odd sub-band; a ladder of n_t chains on distinct walkers (a random permutation), inverse
# temperatures 1.2^-t, each chain holding its own jittered copy of the band's "true" sources (hotter chains
# jitter more; every other chain carries one extra weak source so the sets differ in size).
@dataclass
class TemperTasks:
    N: int
    tasks: dict                  # n_t, chain_begin, n_stage, write_back, k_first   (one entry per task)
    params: np.ndarray           # [n_src_total, 8] all chain sets, read-only
    truth: np.ndarray            # [n_tasks, n_src, 8] the sources the chains scatter around (to build residuals)
    chain_walker: np.ndarray     # [n_chain] int32
    chain_beta: np.ndarray       # [n_chain]
    chain_set_begin: np.ndarray  # [n_chain] int32
    chain_set_n: np.ndarray      # [n_chain] int32
    chain_logu: np.ndarray       # [n_chain] log of the uniform draw of pair (t, t-1); entry t = 0 unused
    max_stage: int


def make_temper_tasks(wl: Workload, N: int, f_lo: float, n_bands: int, n_t: int, n_src: int, stream: int = 0,
                      amp_lo: float = 2e-23, amp_hi: float = 2e-22, jitter: float = 1.0, n_groups: int = 1) -> TemperTasks:
    """n_groups ladders per sub-band on disjoint walkers (tasks are ordered band-major); truth is per band."""
    assert wl.n_walkers >= n_t * n_groups
    g = _rng(wl.config, 200 * _S_BAND + stream + N)
    T = wl.Tobs
    kb0 = int(np.ceil(f_lo * T / N)) * N
    b = 2 * np.arange(n_bands, dtype=np.int64) + 1
    u = g.random((n_bands, n_src, 8))
    tr = np.empty((n_bands, n_src, 8))
    tr[..., 0] = amp_lo * (amp_hi / amp_lo) ** u[..., 0]
    tr[..., 1] = (kb0 + (b[:, None] + 0.1 + 0.8 * u[..., 1]) * N) / T
    tr[..., 2] = (2.0 * u[..., 2] - 1.0) * 1e-16
    tr[..., 3] = 2.0 * np.pi * u[..., 3]
    tr[..., 4] = 1.8 * u[..., 4] - 0.9
    tr[..., 5] = np.pi * u[..., 5]
    tr[..., 6] = 2.0 * np.pi * u[..., 6]
    tr[..., 7] = 1.8 * u[..., 7] - 0.9
    sets, set_begin, set_n, walkers = [], [], [], []
    row = 0
    for i in [ib for ib in range(n_bands) for _ in range(n_groups)]:
        if len(walkers) % n_groups == 0:
            pw = g.permutation(wl.n_walkers).astype(np.int32)
        walkers.append(pw[(len(walkers) % n_groups) * n_t:(len(walkers) % n_groups + 1) * n_t])
        for t in range(n_t):
            z = g.standard_normal((n_src, 8)) * jitter * (1.0 + 0.5 * t)
            s = tr[i].copy()
            s[:, 0] *= 1.0 + 0.01 * z[:, 0]
            s[:, 1] += 3e-10 * z[:, 1]
            s[:, 3] += 0.01 * z[:, 3]
            s[:, 5] += 0.01 * z[:, 5]
            s[:, 6] += 0.005 * z[:, 6]
            if t % 2 == 1:                                   # one extra weak source: sets of different size
                e = tr[i, :1].copy()
                e[0, 0] = 0.05 * amp_lo
                e[0, 1] = (kb0 + (b[i] + g.random()) * N) / T
                s = np.concatenate([s, e])
            sets.append(s)
            set_begin.append(row)
            set_n.append(len(s))
            row += len(s)
    ntask = n_bands * n_groups
    nc = ntask * n_t
    tasks = {"n_t": np.full(ntask, n_t, np.int32), "chain_begin": (np.arange(ntask) * n_t).astype(np.int32),
             "n_stage": np.full(ntask, 3 * N, np.int32), "write_back": np.ones(ntask, np.int32),
             "k_first": np.repeat(kb0 + (b - 1) * N, n_groups)}
    return TemperTasks(N, tasks, np.ascontiguousarray(np.concatenate(sets)), tr, np.concatenate(walkers),
                       np.tile(1.2 ** -np.arange(n_t, dtype=np.float64), ntask), np.asarray(set_begin, np.int32),
                       np.asarray(set_n, np.int32), np.log(g.random(nc)), 3 * N)


# ---------------------------------------------------------------------------------------------------------
# Search-stage batch shape (App. G): per-sub-band fixed-dimension parallel tempering, ~900 sub-bands x
# ~10 temperatures x ~100 walkers, ONE source per walker, every walker of a sub-band evaluated against the same best-fit
# residual of its band; "the priors are modified so that the initial frequency spans its assigned sub-band only" (:712).
# Rows are band-major (all temperatures and walkers of a band are consecutive): the opposite of config 5's geometry -- many
# rows on the same few hundred bins of ONE residual row.
def make_search_stage(n_bands: int = 900, n_temps: int = 10, n_walkers: int = 100, f_lo: float = 3e-4, f_hi: float = 1.5e-2,
                      snr_lo: float = 5.0, snr_hi: float = 30.0, stream: int = 0) -> Workload:
    g = _rng(6, _S_PARAMS + stream)
    k_lo, n_f = band_bins(0.1e-3, 30e-3)
    psd, sc = _psd_rows(6, 1, k_lo, n_f, False)
    # sub-bands spread log-uniformly over [f_lo, f_hi]; a band starts on a multiple of its window length
    fb = np.sort(f_lo * (f_hi / f_lo) ** ((np.arange(n_bands) + g.random(n_bands)) / n_bands))
    Nb = n_bins_for_f0(fb)
    kb = (np.floor(fb * TOBS / Nb) * Nb).astype(np.int64)
    per = n_temps * n_walkers
    B = n_bands * per
    p = _draw_params(g, B, 1e-3, 2e-3)
    band = np.repeat(np.arange(n_bands), per)
    p[:, 1] = (kb[band] + g.random(B) * Nb[band]) / TOBS               # f0 inside its sub-band only
    f = p[:, 1]
    # amplitude from an optimal-SNR draw in [snr_lo, snr_hi] (the search works between the SNR limits 7 -> 5, :718):
    # rho^2 ~ 4/5 amp^2 T_obs x^2 ... is not needed exactly -- scale a reference amplitude by the noise level at f0
    S = instrument_psd(f)
    rho = snr_lo * (snr_hi / snr_lo) ** g.random(B)
    x = 2.0 * np.pi * f * ARMLENGTH / 299792458.0
    p[:, 0] = rho * np.sqrt(S / TOBS) / (np.maximum(np.abs(np.sin(x)), 1e-3) * x) * 0.22
    nb = Nb[band].astype(np.int32)
    return Workload(6, "search_stage", TOBS, DT, k_lo, n_f, 1, psd, None, p, None, np.zeros(B, np.int32), None, ADD, 0, nb,
                    None, sc)
