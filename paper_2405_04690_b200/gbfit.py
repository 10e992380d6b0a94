"""Thin Python binding of the C ABI in include/gbfit.h (argument marshalling only).

Every step of the path (per-source constants, slow part, FFT, window gather, inner products, delta lnL,
scatter-add) runs inside libgbfit.so's CUDA kernels.  torch is used for device memory and streams only;
there is no CPU fallback: if libgbfit.so is missing or does not load, importing this module's `lib()`
raises.  Function names and argument order follow include/gbfit.h (PAPER.md citations are there).
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np
import torch

from . import build as _build

ADD, REMOVE, SWAP = 0, 1, 2
GB_OK, GB_ERR_INVALID, GB_ERR_CUDA, GB_ERR_NOMEM, GB_ERR_ROW = 0, -1, -2, -3, -4

EXPORTS = ("gb_default_config", "gb_create", "gb_destroy", "gb_last_error", "gb_check", "gb_version",
           "gb_launch_count", "gb_measure_fp64_peak", "gb_waveform", "gb_delta_loglike", "gb_residual_update",
           "gb_waveform_host", "gb_delta_loglike_host", "gb_residual_update_host", "gb_band_sweep", "gb_overlap", "gb_temper_sweep",
           "gb_delta_loglike_keep", "gb_residual_update_kept", "gb_band_sweep_generate", "gb_delta_loglike_accept", "gb_delta_loglike_accept_host",
           "gb_band_sweep_static", "gb_scratch_bytes")

BAND_MAX_STAGE = 3072
HOST_ACCEPT_CUTS = (0, 2, 9, 16, 24)    # GB_HOST_ACCEPT_CUTS: chunk c of delta_loglike_accept_host = rows [B a_c / 24, B a_(c+1) / 24)
STATIC_SCRATCH_BYTES = 32 * 1024 * 1024   # GB_STATIC_SCRATCH_BYTES
STATIC_MAX_TASK_BINS = 32768             # GB_STATIC_MAX_TASK_BINS: gb_band_sweep_static takes n_tasks * N up to this
# layout of gb_band_task (include/gbfit.h)
BAND_TASK = np.dtype([("walker", np.int32), ("n_src", np.int32), ("src_begin", np.int32), ("n_prop", np.int32),
                      ("prop_begin", np.int32), ("n_stage", np.int32), ("k_first", np.int64),
                      ("flags", np.int32), ("write_walker", np.int32), ("beta", np.float64)], align=True)
BAND_WRITE_BACK, BAND_SUBTRACT_CURRENT, BAND_WRITE_OTHER = 1, 2, 4


TEMPER_MAX_LADDER = 64
# layout of gb_temper_task (include/gbfit.h)
TEMPER_TASK = np.dtype([("n_t", np.int32), ("chain_begin", np.int32), ("n_stage", np.int32), ("write_back", np.int32),
                        ("k_first", np.int64), ("write_walker", np.int32), ("reserved", np.int32)], align=True)
TEMPER_WRITE_BACK, TEMPER_ODD_EVEN = 1, 2


def pack_temper_tasks(n_t, chain_begin, n_stage, write_back, k_first, write_walker=None) -> np.ndarray:
    """Host array of gb_temper_task records from equal-length columns.  write_walker selects the odd/even cold-chain buffer
    mode of PAPER.md:354-362 (GB_TEMPER_ODD_EVEN): the row that receives exchanges with the cold chain."""
    t = np.zeros(len(n_t), TEMPER_TASK)
    for key, val in (("n_t", n_t), ("chain_begin", chain_begin), ("n_stage", n_stage), ("k_first", k_first)):
        t[key] = val
    t["write_back"] = (np.asarray(write_back) != 0).astype(np.int32)
    if write_walker is not None:
        t["write_back"] |= TEMPER_ODD_EVEN
        t["write_walker"] = write_walker
    return t


def pack_band_tasks(walker, n_src, src_begin, n_prop, prop_begin, n_stage, k_first, write_back, beta,
                    subtract_current=None, write_walker=None) -> np.ndarray:
    """Host array of gb_band_task records from equal-length columns (upload it as bytes:
    torch.from_numpy(t.view(np.uint8))).  subtract_current / write_walker select the odd/even cold-chain buffer mode
    of PAPER.md:354-362 (GB_BAND_SUBTRACT_CURRENT, GB_BAND_WRITE_OTHER)."""
    t = np.zeros(len(walker), BAND_TASK)
    for key, val in (("walker", walker), ("n_src", n_src), ("src_begin", src_begin), ("n_prop", n_prop),
                     ("prop_begin", prop_begin), ("n_stage", n_stage), ("k_first", k_first), ("beta", beta)):
        t[key] = val
    flags = BAND_WRITE_BACK * (np.asarray(write_back) != 0).astype(np.int32)
    if subtract_current is not None:
        flags |= BAND_SUBTRACT_CURRENT * (np.asarray(subtract_current) != 0).astype(np.int32)
    if write_walker is not None:
        flags |= BAND_WRITE_OTHER
        t["write_walker"] = write_walker
    t["flags"] = flags
    return t


class GbConfig(C.Structure):
    _fields_ = [("Tobs", C.c_double), ("dt", C.c_double), ("armlength", C.c_double), ("au", C.c_double),
                ("year", C.c_double), ("kappa", C.c_double), ("lambda0", C.c_double),
                ("device", C.c_int32), ("reserved", C.c_int32)]


class GbData(C.Structure):
    _fields_ = [("resid", C.c_void_p), ("psd", C.c_void_p), ("walker_psd", C.c_void_p),
                ("k_lo", C.c_int64), ("n_f", C.c_int64),
                ("n_walkers", C.c_int32), ("n_psd", C.c_int32), ("psd_is_inverse", C.c_int32),
                ("reserved", C.c_int32)]


class GbStretch(C.Structure):   # gb_stretch (include/gbfit.h)
    _fields_ = [("seed", C.c_uint64), ("sweep", C.c_uint32), ("n_friends", C.c_int32), ("group", C.c_void_p),
                ("n_group", C.c_int64), ("stretch_a", C.c_double), ("lo", C.c_double * 8), ("hi", C.c_double * 8),
                ("periodic", C.c_int32 * 8)]


class Stretch:
    """Inputs of the in-loop proposal step of gb_band_sweep_generate: Philox seed / sweep, the stationary group as a CUDA
    tensor [n_group, 8] sorted by f0 ascending (the caller sorts it), n_friends, stretch scale a, prior box, periodic flags."""

    def __init__(self, seed: int, sweep: int, group: torch.Tensor, n_friends: int, lo, hi, periodic, stretch_a: float = 2.0):
        self.seed, self.sweep, self.group, self.n_friends = int(seed), int(sweep), group, int(n_friends)
        self.lo, self.hi, self.periodic, self.stretch_a = [float(x) for x in lo], [float(x) for x in hi], \
            [int(x) for x in periodic], float(stretch_a)
        if len(self.lo) != 8 or len(self.hi) != 8 or len(self.periodic) != 8:
            raise ValueError("lo, hi, periodic must have 8 entries")

    def c(self, device):
        g = _dev_ptr(self.group, torch.float64, device, "group")
        if self.group.dim() != 2 or self.group.shape[1] != 8:
            raise ValueError("group must be [n_group, 8]")
        return C.byref(GbStretch(self.seed, self.sweep, self.n_friends, g, int(self.group.shape[0]), self.stretch_a,
                                 (C.c_double * 8)(*self.lo), (C.c_double * 8)(*self.hi), (C.c_int32 * 8)(*self.periodic)))


class GbError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"gbfit error {code}: {msg}")
        self.code = code


_lib = None


def lib_path() -> str:
    return _build.LIB


def lib() -> C.CDLL:
    """Load libgbfit.so (built in-tree by paper_2405_04690_b200.build).  Fails loudly when absent."""
    global _lib
    if _lib is None:
        path = lib_path()
        if not os.path.exists(path):
            raise ImportError(f"{path} is missing: run `python -m paper_2405_04690_b200.build` "
                              "(the GB hot path has no CPU or PyTorch fallback)")
        L = C.CDLL(path)
        vp, i64, i32, ci = C.c_void_p, C.c_int64, C.c_int32, C.c_int
        L.gb_default_config.argtypes = [C.POINTER(GbConfig)]
        L.gb_default_config.restype = None
        L.gb_create.argtypes = [C.POINTER(GbConfig), C.POINTER(vp)]
        L.gb_create.restype = ci
        L.gb_destroy.argtypes = [vp]
        L.gb_destroy.restype = None
        L.gb_last_error.argtypes = [vp]
        L.gb_last_error.restype = C.c_char_p
        L.gb_check.argtypes = [vp, vp]
        L.gb_check.restype = ci
        L.gb_version.argtypes = []
        L.gb_version.restype = C.c_char_p
        L.gb_launch_count.argtypes = [vp]
        L.gb_launch_count.restype = i64
        L.gb_scratch_bytes.argtypes = [vp]
        L.gb_scratch_bytes.restype = i64
        L.gb_measure_fp64_peak.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_double, vp]
        L.gb_measure_fp64_peak.restype = ci
        wf = [vp, vp, i64, ci, vp, ci, vp, vp, vp]
        dl = [vp, C.POINTER(GbData), vp, vp, vp, vp, ci, ci, vp, i64, vp, vp, vp]
        ru = [vp, C.POINTER(GbData), vp, vp, vp, vp, ci, vp, ci, vp, i64, vp]
        L.gb_band_sweep.argtypes = [vp, C.POINTER(GbData), vp, i64, ci, ci, vp, vp, vp, vp, vp, vp, vp, vp]
        L.gb_band_sweep.restype = ci
        L.gb_band_sweep_static.argtypes = L.gb_band_sweep.argtypes
        L.gb_band_sweep_static.restype = ci
        L.gb_band_sweep_generate.argtypes = [vp, C.POINTER(GbData), vp, i64, ci, ci, vp, C.POINTER(GbStretch), vp, vp, vp, vp,
                                             vp, vp, vp]
        L.gb_band_sweep_generate.restype = ci
        L.gb_overlap.argtypes = [vp, C.POINTER(GbData), vp, vp, vp, ci, vp, i64, vp, vp, vp]
        L.gb_overlap.restype = ci
        L.gb_delta_loglike_keep.argtypes = [vp, C.POINTER(GbData), vp, vp, vp, vp, ci, ci, vp, i64, i64, vp, vp, vp]
        L.gb_delta_loglike_keep.restype = ci
        L.gb_delta_loglike_accept.argtypes = [vp, C.POINTER(GbData), vp, vp, vp, vp, ci, ci, vp, i64, vp, vp, vp, i64, ci, vp,
                                              vp, vp, vp]
        L.gb_delta_loglike_accept.restype = ci
        L.gb_delta_loglike_accept_host.argtypes = L.gb_delta_loglike_accept.argtypes
        L.gb_delta_loglike_accept_host.restype = ci
        L.gb_residual_update_kept.argtypes = [vp, C.POINTER(GbData), vp, ci, vp]
        L.gb_residual_update_kept.restype = ci
        L.gb_temper_sweep.argtypes = [vp, C.POINTER(GbData), vp, i64, ci, ci, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
        L.gb_temper_sweep.restype = ci
        for name, sig in (("gb_waveform", wf), ("gb_waveform_host", wf), ("gb_delta_loglike", dl),
                          ("gb_delta_loglike_host", dl), ("gb_residual_update", ru),
                          ("gb_residual_update_host", ru)):
            fn = getattr(L, name)
            fn.argtypes = sig
            fn.restype = ci
        _lib = L
    return _lib


def version() -> str:
    return lib().gb_version().decode()


# ----------------------------------------------------------------------------------------- marshalling
def _dev_ptr(t: Optional[torch.Tensor], dtype, device, name: str):
    if t is None:
        return None
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError(f"{name} must be a CUDA tensor")
    if t.device != device:
        raise ValueError(f"{name} is on {t.device}, context is on {device}")
    dts = dtype if isinstance(dtype, tuple) else (dtype,)
    if t.dtype not in dts:
        raise TypeError(f"{name} must have dtype {dts}, got {t.dtype}")
    if not t.is_contiguous():
        raise ValueError(f"{name} must be contiguous")
    return C.c_void_p(t.data_ptr())


def _host_ptr(a, dtype, name: str):
    """numpy array or CPU torch tensor (pinned or not) -> (void*, keepalive)."""
    if a is None:
        return None, None
    if isinstance(a, torch.Tensor):
        if a.is_cuda:
            raise TypeError(f"{name} must be a HOST buffer")
        if not a.is_contiguous():
            raise ValueError(f"{name} must be contiguous")
        want = {np.float64: torch.float64, np.int32: torch.int32, np.int8: torch.int8, np.uint8: torch.uint8,
                np.int64: torch.int64, np.complex128: torch.complex128}[dtype]
        if a.dtype != want:
            raise TypeError(f"{name} must have dtype {want}, got {a.dtype}")
        return C.c_void_p(a.data_ptr()), a
    arr = np.ascontiguousarray(a, dtype=dtype)
    return C.c_void_p(arr.ctypes.data), arr


def _stream_ptr(stream, device):
    if stream is None:
        stream = torch.cuda.current_stream(device)
    if isinstance(stream, torch.cuda.Stream):
        return C.c_void_p(stream.cuda_stream)
    return C.c_void_p(int(stream))


class Data:
    """Device-resident residuals and PSDs of the walkers (gb_data of include/gbfit.h).

    resid: CUDA complex128 [n_walkers, 2, n_f] (or float64 [n_walkers, 2, n_f, 2]); modified in place by
    residual_update.  psd: CUDA float64 [n_psd, 2, n_f].  walker_psd: CUDA int32 [n_walkers] or None.
    """

    def __init__(self, resid: torch.Tensor, psd: torch.Tensor, k_lo: int,
                 walker_psd: Optional[torch.Tensor] = None, psd_is_inverse: bool = False):
        if resid.dtype == torch.complex128:
            if resid.dim() != 3 or resid.shape[1] != 2:
                raise ValueError("resid must be [n_walkers, 2, n_f] complex128")
        elif resid.dtype == torch.float64:
            if resid.dim() != 4 or resid.shape[1] != 2 or resid.shape[3] != 2:
                raise ValueError("resid must be [n_walkers, 2, n_f, 2] float64")
        else:
            raise TypeError("resid must be complex128 or float64")
        if psd.dim() != 3 or psd.shape[1] != 2 or psd.shape[2] != resid.shape[2]:
            raise ValueError("psd must be [n_psd, 2, n_f] float64")
        dev = resid.device
        self.resid, self.psd, self.walker_psd = resid, psd, walker_psd
        self.k_lo, self.n_f = int(k_lo), int(resid.shape[2])
        self.n_walkers, self.n_psd = int(resid.shape[0]), int(psd.shape[0])
        if walker_psd is None and self.n_psd not in (1, self.n_walkers):
            raise ValueError("walker_psd is required when n_psd is neither 1 nor n_walkers")
        self.psd_is_inverse = bool(psd_is_inverse)
        self.device = dev
        self._c = GbData(_dev_ptr(resid, (torch.complex128, torch.float64), dev, "resid"),
                         _dev_ptr(psd, torch.float64, dev, "psd"),
                         _dev_ptr(walker_psd, torch.int32, dev, "walker_psd"),
                         self.k_lo, self.n_f, self.n_walkers, self.n_psd, int(self.psd_is_inverse), 0)

    def c(self):
        return C.byref(self._c)

    @classmethod
    def psd_only(cls, psd: torch.Tensor, k_lo: int, psd_is_inverse: bool = False) -> "Data":
        """A view without residuals, for gb_overlap: psd CUDA float64 [n_psd, 2, n_f]."""
        if psd.dim() != 3 or psd.shape[1] != 2:
            raise ValueError("psd must be [n_psd, 2, n_f] float64")
        self = cls.__new__(cls)
        self.resid, self.psd, self.walker_psd = None, psd, None
        self.k_lo, self.n_f = int(k_lo), int(psd.shape[2])
        self.n_walkers, self.n_psd = 0, int(psd.shape[0])
        self.psd_is_inverse = bool(psd_is_inverse)
        self.device = psd.device
        self._c = GbData(None, _dev_ptr(psd, torch.float64, psd.device, "psd"), None, self.k_lo, self.n_f, 0,
                         self.n_psd, int(self.psd_is_inverse), 0)
        return self


class Context:
    """gb_ctx: orbit tables, twiddles and scratch on one device."""

    def __init__(self, device: int = 0, **cfg):
        L = lib()
        c = GbConfig()
        L.gb_default_config(C.byref(c))
        for k, v in cfg.items():
            if not hasattr(c, k) or k in ("device", "reserved"):
                raise TypeError(f"unknown gb_config field {k}")
            setattr(c, k, float(v))
        c.device = int(device)
        self.config = c
        self.device = torch.device("cuda", int(device))
        self._h = C.c_void_p()
        rc = L.gb_create(C.byref(c), C.byref(self._h))
        if rc != GB_OK:
            msg = L.gb_last_error(self._h).decode() if self._h else "gb_create failed"
            if self._h:
                L.gb_destroy(self._h)
                self._h = C.c_void_p()
            raise GbError(rc, msg)

    def close(self):
        if getattr(self, "_h", None):
            lib().gb_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def _ok(self, rc: int):
        if rc != GB_OK:
            raise GbError(rc, lib().gb_last_error(self._h).decode())

    def last_error(self) -> str:
        return lib().gb_last_error(self._h).decode()

    def launch_count(self) -> int:
        return int(lib().gb_launch_count(self._h))

    def scratch_bytes(self) -> int:
        """gb_scratch_bytes: device scratch the context holds right now."""
        return int(lib().gb_scratch_bytes(self._h))

    def measure_fp64_peak(self, clock_mhz: float = 0.0, stream=None):
        """Diagnostic: sustained DFMA rate of the device -> (TFLOP/s, DFMA lanes per SM per clock at clock_mhz)."""
        tf, lanes = C.c_double(0.0), C.c_double(0.0)
        self._ok(lib().gb_measure_fp64_peak(self._h, C.byref(tf), C.byref(lanes), C.c_double(clock_mhz),
                                            _stream_ptr(stream, self.device)))
        return float(tf.value), float(lanes.value)

    def check(self, stream=None):
        """Synchronise the stream and raise if any row of an earlier call was invalid."""
        self._ok(lib().gb_check(self._h, _stream_ptr(stream, self.device)))

    # ------------------------------------------------------------------------------- device forms
    def waveform(self, params: torch.Tensor, N: int = 0, n_bins: Optional[torch.Tensor] = None,
                 Nmax: Optional[int] = None, out: Optional[torch.Tensor] = None,
                 kmin_out: Optional[torch.Tensor] = None, stream=None):
        """gb_waveform: returns (AE [B, 2, Nmax] complex128, kmin [B] int64), both CUDA tensors."""
        dev = self.device
        B = int(params.shape[0])
        if Nmax is None:
            Nmax = int(N) if n_bins is None else 1024
        if out is None:
            out = torch.zeros((B, 2, Nmax), dtype=torch.complex128, device=dev)
        if kmin_out is None:
            kmin_out = torch.empty((B,), dtype=torch.int64, device=dev)
        self._ok(lib().gb_waveform(self._h, _dev_ptr(params, torch.float64, dev, "params"), B, int(N),
                                   _dev_ptr(n_bins, torch.int32, dev, "n_bins"), int(Nmax),
                                   _dev_ptr(out, (torch.complex128, torch.float64), dev, "out"),
                                   _dev_ptr(kmin_out, torch.int64, dev, "kmin_out"),
                                   _stream_ptr(stream, dev)))
        return out, kmin_out

    def delta_loglike(self, data: Data, params_new: Optional[torch.Tensor], params_old: Optional[torch.Tensor],
                      walker_index: torch.Tensor, move: Optional[torch.Tensor] = None, move_all: int = ADD,
                      N: int = 0, n_bins: Optional[torch.Tensor] = None, out: Optional[torch.Tensor] = None,
                      aux: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
        """gb_delta_loglike: returns dlnL [B] float64 (CUDA)."""
        dev = self.device
        B = int(walker_index.shape[0])
        if out is None:
            out = torch.empty((B,), dtype=torch.float64, device=dev)
        self._ok(lib().gb_delta_loglike(self._h, data.c(), _dev_ptr(params_new, torch.float64, dev, "params_new"),
                                        _dev_ptr(params_old, torch.float64, dev, "params_old"),
                                        _dev_ptr(walker_index, torch.int32, dev, "walker_index"),
                                        _dev_ptr(move, torch.int8, dev, "move"), int(move_all), int(N),
                                        _dev_ptr(n_bins, torch.int32, dev, "n_bins"), B,
                                        _dev_ptr(out, torch.float64, dev, "out"),
                                        _dev_ptr(aux, torch.float64, dev, "aux"), _stream_ptr(stream, dev)))
        return out

    def delta_loglike_keep(self, data: Data, params_new: Optional[torch.Tensor], params_old: Optional[torch.Tensor],
                           walker_index: torch.Tensor, move: Optional[torch.Tensor] = None, move_all: int = ADD,
                           N: int = 0, n_bins: Optional[torch.Tensor] = None, sum_n_bins: int = 0,
                           out: Optional[torch.Tensor] = None, aux: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
        """gb_delta_loglike_keep: delta lnL of ADD / REMOVE rows; the windows stay in the context for residual_update_kept.
        sum_n_bins = int(n_bins.sum()) when n_bins is given."""
        dev = self.device
        B = int(walker_index.shape[0])
        if out is None:
            out = torch.empty((B,), dtype=torch.float64, device=dev)
        self._ok(lib().gb_delta_loglike_keep(self._h, data.c(), _dev_ptr(params_new, torch.float64, dev, "params_new"),
                                             _dev_ptr(params_old, torch.float64, dev, "params_old"),
                                             _dev_ptr(walker_index, torch.int32, dev, "walker_index"),
                                             _dev_ptr(move, torch.int8, dev, "move"), int(move_all), int(N),
                                             _dev_ptr(n_bins, torch.int32, dev, "n_bins"), B, int(sum_n_bins),
                                             _dev_ptr(out, torch.float64, dev, "out"),
                                             _dev_ptr(aux, torch.float64, dev, "aux"), _stream_ptr(stream, dev)))
        return out

    def delta_loglike_accept(self, data: Data, params_new: Optional[torch.Tensor], params_old: Optional[torch.Tensor],
                             walker_index: torch.Tensor, logu: torch.Tensor, logq: Optional[torch.Tensor] = None,
                             beta: Optional[torch.Tensor] = None, move: Optional[torch.Tensor] = None, move_all: int = ADD,
                             N: int = 0, n_bins: Optional[torch.Tensor] = None, store_bins: int = 0, apply: int = 1,
                             out: Optional[torch.Tensor] = None, aux: Optional[torch.Tensor] = None,
                             accepted_out: Optional[torch.Tensor] = None, stream=None):
        """gb_delta_loglike_accept: delta lnL of every ADD / REMOVE row against one snapshot, accepted iff
        beta dlnL + logq >= logu, then (apply 1: fused, 2: separate launch) the update by the accepted rows;
        apply 0 keeps the accepted windows for residual_update_kept(data, None).  Returns (dlnL, accepted uint8)."""
        dev = self.device
        B = int(walker_index.shape[0])
        if out is None:
            out = torch.empty((B,), dtype=torch.float64, device=dev)
        if accepted_out is None:
            accepted_out = torch.zeros((B,), dtype=torch.uint8, device=dev)
        self._ok(lib().gb_delta_loglike_accept(self._h, data.c(), _dev_ptr(params_new, torch.float64, dev, "params_new"),
                                               _dev_ptr(params_old, torch.float64, dev, "params_old"),
                                               _dev_ptr(walker_index, torch.int32, dev, "walker_index"),
                                               _dev_ptr(move, torch.int8, dev, "move"), int(move_all), int(N),
                                               _dev_ptr(n_bins, torch.int32, dev, "n_bins"), B,
                                               _dev_ptr(logq, torch.float64, dev, "logq"),
                                               _dev_ptr(logu, torch.float64, dev, "logu"),
                                               _dev_ptr(beta, torch.float64, dev, "beta"), int(store_bins), int(apply),
                                               _dev_ptr(out, torch.float64, dev, "out"),
                                               _dev_ptr(aux, torch.float64, dev, "aux"),
                                               _dev_ptr(accepted_out, torch.uint8, dev, "accepted_out"),
                                               _stream_ptr(stream, dev)))
        return out, accepted_out

    def residual_update_kept(self, data: Data, accepted: Optional[torch.Tensor] = None, negate: bool = False,
                             stream=None) -> None:
        """gb_residual_update_kept: scatter the accepted rows of the preceding delta_loglike_keep call."""
        dev = self.device
        self._ok(lib().gb_residual_update_kept(self._h, data.c(), _dev_ptr(accepted, torch.uint8, dev, "accepted"),
                                               int(bool(negate)), _stream_ptr(stream, dev)))

    def residual_update(self, data: Data, params_new: Optional[torch.Tensor], params_old: Optional[torch.Tensor],
                        walker_index: torch.Tensor, move: Optional[torch.Tensor] = None, move_all: int = ADD,
                        accepted: Optional[torch.Tensor] = None, N: int = 0,
                        n_bins: Optional[torch.Tensor] = None, stream=None) -> None:
        """gb_residual_update: scatter accepted rows into data.resid in place."""
        dev = self.device
        B = int(walker_index.shape[0])
        self._ok(lib().gb_residual_update(self._h, data.c(), _dev_ptr(params_new, torch.float64, dev, "params_new"),
                                          _dev_ptr(params_old, torch.float64, dev, "params_old"),
                                          _dev_ptr(walker_index, torch.int32, dev, "walker_index"),
                                          _dev_ptr(move, torch.int8, dev, "move"), int(move_all),
                                          _dev_ptr(accepted, torch.uint8, dev, "accepted"), int(N),
                                          _dev_ptr(n_bins, torch.int32, dev, "n_bins"), B,
                                          _stream_ptr(stream, dev)))

    def overlap(self, data: Data, params_a: torch.Tensor, params_c: torch.Tensor,
                psd_row: Optional[torch.Tensor] = None, N: int = 0, n_bins: Optional[torch.Tensor] = None,
                out: Optional[torch.Tensor] = None, aux: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
        """gb_overlap: normalised overlap [B] float64 (CUDA); aux [B, 2] receives <a|a>, <c|c> when given."""
        dev = self.device
        B = int(params_a.shape[0])
        if out is None:
            out = torch.empty((B,), dtype=torch.float64, device=dev)
        self._ok(lib().gb_overlap(self._h, data.c(), _dev_ptr(params_a, torch.float64, dev, "params_a"),
                                  _dev_ptr(params_c, torch.float64, dev, "params_c"),
                                  _dev_ptr(psd_row, torch.int32, dev, "psd_row"), int(N),
                                  _dev_ptr(n_bins, torch.int32, dev, "n_bins"), B,
                                  _dev_ptr(out, torch.float64, dev, "out"),
                                  _dev_ptr(aux, torch.float64, dev, "aux"), _stream_ptr(stream, dev)))
        return out

    def temper_sweep(self, data: Data, tasks: torch.Tensor, N: int, max_stage: int, params: torch.Tensor,
                     chain_walker: torch.Tensor, chain_beta: torch.Tensor, chain_set_begin: torch.Tensor,
                     chain_set_n: torch.Tensor, chain_logu: torch.Tensor, stream=None):
        """gb_temper_sweep (Algorithm 2, Eq. D2): `tasks` is a CUDA uint8 tensor of packed gb_temper_task records
        (pack_temper_tasks).  Returns (perm int32, accepted uint8, dlnl [n_chain, 2] float64), CUDA tensors;
        data.resid is updated in place for accepted exchanges of tasks with write_back."""
        dev = self.device
        n_tasks = int(tasks.numel() // TEMPER_TASK.itemsize)
        nc = int(chain_walker.shape[0])
        perm = torch.zeros((nc,), dtype=torch.int32, device=dev)
        acc = torch.zeros((nc,), dtype=torch.uint8, device=dev)
        dl = torch.zeros((nc, 2), dtype=torch.float64, device=dev)
        self._ok(lib().gb_temper_sweep(self._h, data.c(), _dev_ptr(tasks, torch.uint8, dev, "tasks"), n_tasks, int(N),
                                       int(max_stage), _dev_ptr(params, torch.float64, dev, "params"),
                                       _dev_ptr(chain_walker, torch.int32, dev, "chain_walker"),
                                       _dev_ptr(chain_beta, torch.float64, dev, "chain_beta"),
                                       _dev_ptr(chain_set_begin, torch.int32, dev, "chain_set_begin"),
                                       _dev_ptr(chain_set_n, torch.int32, dev, "chain_set_n"),
                                       _dev_ptr(chain_logu, torch.float64, dev, "chain_logu"),
                                       _dev_ptr(perm, torch.int32, dev, "perm"), _dev_ptr(acc, torch.uint8, dev, "acc"),
                                       _dev_ptr(dl, torch.float64, dev, "dl"), _stream_ptr(stream, dev)))
        return perm, acc, dl

    def band_sweep(self, data: Data, tasks: torch.Tensor, N: int, max_stage: int, params: torch.Tensor,
                   prop_k: torch.Tensor, prop_params: torch.Tensor, prop_logq: torch.Tensor, prop_logu: torch.Tensor,
                   accepted_out: Optional[torch.Tensor] = None, dlnL_out: Optional[torch.Tensor] = None, stream=None):
        """gb_band_sweep (Algorithm 1): `tasks` is a CUDA uint8 tensor holding packed gb_band_task records
        (pack_band_tasks); params [n_src_total, 8] and data.resid are updated in place.
        Returns (accepted [n_prop_total] uint8, dlnL [n_prop_total] float64), CUDA tensors."""
        dev = self.device
        n_tasks = int(tasks.numel() // BAND_TASK.itemsize)
        P = int(prop_k.shape[0])
        if accepted_out is None:
            accepted_out = torch.zeros((P,), dtype=torch.uint8, device=dev)
        if dlnL_out is None:
            dlnL_out = torch.zeros((P,), dtype=torch.float64, device=dev)
        self._ok(lib().gb_band_sweep(self._h, data.c(), _dev_ptr(tasks, torch.uint8, dev, "tasks"), n_tasks, int(N),
                                     int(max_stage), _dev_ptr(params, torch.float64, dev, "params"),
                                     _dev_ptr(prop_k, torch.int32, dev, "prop_k"),
                                     _dev_ptr(prop_params, torch.float64, dev, "prop_params"),
                                     _dev_ptr(prop_logq, torch.float64, dev, "prop_logq"),
                                     _dev_ptr(prop_logu, torch.float64, dev, "prop_logu"),
                                     _dev_ptr(accepted_out, torch.uint8, dev, "accepted_out"),
                                     _dev_ptr(dlnL_out, torch.float64, dev, "dlnL_out"), _stream_ptr(stream, dev)))
        return accepted_out, dlnL_out

    def band_sweep_static(self, data: Data, tasks: torch.Tensor, N: int, max_stage: int, params: torch.Tensor,
                          prop_k: torch.Tensor, prop_params: torch.Tensor, prop_logq: torch.Tensor, prop_logu: torch.Tensor,
                          accepted_out: torch.Tensor, dlnL_out: torch.Tensor, stream=None):
        """gb_band_sweep_static: gb_band_sweep with the kernel's scratch in the library's static device array; the call
        allocates nothing (the caller passes both outputs), n_tasks * N <= STATIC_MAX_TASK_BINS, and calls that overlap on
        the GPU race on the shared array.  Returns (accepted_out, dlnL_out)."""
        dev = self.device
        n_tasks = int(tasks.numel() // BAND_TASK.itemsize)
        self._ok(lib().gb_band_sweep_static(self._h, data.c(), _dev_ptr(tasks, torch.uint8, dev, "tasks"), n_tasks, int(N),
                                            int(max_stage), _dev_ptr(params, torch.float64, dev, "params"),
                                            _dev_ptr(prop_k, torch.int32, dev, "prop_k"),
                                            _dev_ptr(prop_params, torch.float64, dev, "prop_params"),
                                            _dev_ptr(prop_logq, torch.float64, dev, "prop_logq"),
                                            _dev_ptr(prop_logu, torch.float64, dev, "prop_logu"),
                                            _dev_ptr(accepted_out, torch.uint8, dev, "accepted_out"),
                                            _dev_ptr(dlnL_out, torch.float64, dev, "dlnL_out"), _stream_ptr(stream, dev)))
        return accepted_out, dlnL_out

    def band_sweep_generate(self, data: Data, tasks: torch.Tensor, N: int, max_stage: int, params: torch.Tensor,
                            stretch: "Stretch", n_prop_total: int, stream=None):
        """gb_band_sweep_generate (Algorithm 1 with the proposal step inside the loop): params and
        data.resid are updated in place.  Returns CUDA tensors (accepted uint8, dlnL, k int32, theta' [P, 8], logq, logu)
        over all P = n_prop_total proposal rows."""
        dev = self.device
        n_tasks = int(tasks.numel() // BAND_TASK.itemsize)
        P = int(n_prop_total)
        acc = torch.zeros((P,), dtype=torch.uint8, device=dev)
        dl = torch.zeros((P,), dtype=torch.float64, device=dev)
        k = torch.zeros((P,), dtype=torch.int32, device=dev)
        pp = torch.zeros((P, 8), dtype=torch.float64, device=dev)
        lq = torch.zeros((P,), dtype=torch.float64, device=dev)
        lu = torch.zeros((P,), dtype=torch.float64, device=dev)
        self._ok(lib().gb_band_sweep_generate(self._h, data.c(), _dev_ptr(tasks, torch.uint8, dev, "tasks"), n_tasks, int(N),
                                              int(max_stage), _dev_ptr(params, torch.float64, dev, "params"),
                                              stretch.c(dev), _dev_ptr(k, torch.int32, dev, "k_out"),
                                              _dev_ptr(pp, torch.float64, dev, "params_out"),
                                              _dev_ptr(lq, torch.float64, dev, "logq_out"),
                                              _dev_ptr(lu, torch.float64, dev, "logu_out"),
                                              _dev_ptr(acc, torch.uint8, dev, "accepted_out"),
                                              _dev_ptr(dl, torch.float64, dev, "dlnL_out"), _stream_ptr(stream, dev)))
        return acc, dl, k, pp, lq, lu

    # --------------------------------------------------------------------------------- host forms
    def waveform_host(self, params, N: int = 0, n_bins=None, Nmax: Optional[int] = None, out=None,
                      kmin_out=None, stream=None):
        """gb_waveform_host: HOST params in, HOST (AE, kmin) out (numpy unless buffers are given)."""
        p, k0 = _host_ptr(params, np.float64, "params")
        B = int(np.prod(k0.shape) // 8)
        nb, k1 = _host_ptr(n_bins, np.int32, "n_bins")
        if Nmax is None:
            Nmax = int(N) if n_bins is None else 1024
        if out is None:
            out = np.zeros((B, 2, Nmax), np.complex128)
        if kmin_out is None:
            kmin_out = np.zeros((B,), np.int64)
        o, k2 = _host_ptr(out, np.complex128, "out")
        km, k3 = _host_ptr(kmin_out, np.int64, "kmin_out")
        self._ok(lib().gb_waveform_host(self._h, p, B, int(N), nb, int(Nmax), o, km,
                                        _stream_ptr(stream, self.device)))
        return k2, k3

    def delta_loglike_host(self, data: Data, params_new, params_old, walker_index, move=None,
                           move_all: int = ADD, N: int = 0, n_bins=None, out=None, aux=None, stream=None):
        """gb_delta_loglike_host: HOST proposal arrays in, HOST dlnL out; `data` stays on the device."""
        pn, k0 = _host_ptr(params_new, np.float64, "params_new")
        po, k1 = _host_ptr(params_old, np.float64, "params_old")
        w, k2 = _host_ptr(walker_index, np.int32, "walker_index")
        B = int(k2.shape[0])
        mv, k3 = _host_ptr(move, np.int8, "move")
        nb, k4 = _host_ptr(n_bins, np.int32, "n_bins")
        if out is None:
            out = np.zeros((B,), np.float64)
        o, k5 = _host_ptr(out, np.float64, "out")
        ax, k6 = _host_ptr(aux, np.float64, "aux")
        self._ok(lib().gb_delta_loglike_host(self._h, data.c(), pn, po, w, mv, int(move_all), int(N), nb, B, o, ax,
                                             _stream_ptr(stream, self.device)))
        return k5

    def delta_loglike_accept_host(self, data: Data, params_new, params_old, walker_index, logu, logq=None, beta=None,
                                  move=None, move_all: int = ADD, N: int = 0, n_bins=None, store_bins: int = 0, apply: int = 1,
                                  out=None, accepted_out=None, stream=None):
        """gb_delta_loglike_accept_host: HOST proposal arrays in, HOST (dlnL, accepted) out; `data` stays on the device."""
        pn, k0 = _host_ptr(params_new, np.float64, "params_new")
        po, k1 = _host_ptr(params_old, np.float64, "params_old")
        w, k2 = _host_ptr(walker_index, np.int32, "walker_index")
        B = int(k2.shape[0])
        mv, k3 = _host_ptr(move, np.int8, "move")
        nb, k4 = _host_ptr(n_bins, np.int32, "n_bins")
        lu, k5 = _host_ptr(logu, np.float64, "logu")
        lq, k6 = _host_ptr(logq, np.float64, "logq")
        bt, k7 = _host_ptr(beta, np.float64, "beta")
        if out is None:
            out = np.zeros((B,), np.float64)
        if accepted_out is None:
            accepted_out = np.zeros((B,), np.uint8)
        o, k8 = _host_ptr(out, np.float64, "out")
        a, k9 = _host_ptr(accepted_out, np.uint8, "accepted_out")
        self._ok(lib().gb_delta_loglike_accept_host(self._h, data.c(), pn, po, w, mv, int(move_all), int(N), nb, B, lq, lu, bt,
                                                    int(store_bins), int(apply), o, None, a,
                                                    _stream_ptr(stream, self.device)))
        return k8, k9

    def residual_update_host(self, data: Data, params_new, params_old, walker_index, move=None,
                             move_all: int = ADD, accepted=None, N: int = 0, n_bins=None, stream=None) -> None:
        """gb_residual_update_host: HOST proposal arrays in; data.resid (device) updated in place."""
        pn, k0 = _host_ptr(params_new, np.float64, "params_new")
        po, k1 = _host_ptr(params_old, np.float64, "params_old")
        w, k2 = _host_ptr(walker_index, np.int32, "walker_index")
        B = int(k2.shape[0])
        mv, k3 = _host_ptr(move, np.int8, "move")
        acc, k4 = _host_ptr(accepted, np.uint8, "accepted")
        nb, k5 = _host_ptr(n_bins, np.int32, "n_bins")
        self._ok(lib().gb_residual_update_host(self._h, data.c(), pn, po, w, mv, int(move_all), acc, int(N), nb, B,
                                               _stream_ptr(stream, self.device)))
