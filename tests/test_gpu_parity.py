"""Parity of the CUDA path (through the C ABI) with the CPU oracle, element by element, on the same seeded
inputs.  Tolerances are the north_star's: waveform bins <= 1e-9 of the source's peak bin (DESIGN.md reading
S16), delta lnL <= 1e-6 absolute, window start bins bit-exact.  All tests need a B200: -m gpu.
"""
import numpy as np
import pytest

from gb_inputs import make_workload, n_bins_for_f0

pytestmark = pytest.mark.gpu

TOL_WF = 1e-9      # max_j |dA_j| / max_j |A_j| per source and channel
TOL_DLNL = 1e-6    # absolute


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu-marked parity tests must run on a B200 box")
    return torch


@pytest.fixture(scope="module")
def gb(torch_cuda):
    from paper_2405_04690_b200 import gbfit
    ctx = gbfit.Context(0)
    yield gbfit, ctx
    ctx.close()


def dev(torch, a, dtype=None):
    return None if a is None else torch.as_tensor(np.ascontiguousarray(a), dtype=dtype).to("cuda:0")


def upload(torch, gbfit, wl, resid, **kw):
    d_resid = dev(torch, resid)
    return gbfit.Data(d_resid, dev(torch, wl.psd), wl.k_lo,
                      walker_psd=dev(torch, wl.walker_psd), **kw), d_resid


def wf_err(got, ref, n_bins=None):
    """max over sources/channels of max_j |d| / max_j |ref| on each row's own N bins."""
    peak = np.abs(ref).max(axis=2, keepdims=True)
    err = np.abs(got - ref) / peak
    if n_bins is not None:
        mask = np.arange(ref.shape[2])[None, None, :] < np.asarray(n_bins)[:, None, None]
        err = np.where(mask, err, 0.0)
    return float(err.max())


def gpu_dlnl(torch, gbfit, ctx, wl, data, aux=False):
    B = wl.B
    d_aux = torch.zeros((B, 2), dtype=torch.float64, device="cuda:0") if aux else None
    out = ctx.delta_loglike(data, dev(torch, wl.params_new), dev(torch, wl.params_old),
                            dev(torch, wl.walker_index), move=dev(torch, wl.move), move_all=wl.move_all,
                            N=wl.N, n_bins=dev(torch, wl.n_bins), aux=d_aux)
    ctx.check()
    return (out.cpu().numpy(), d_aux.cpu().numpy()) if aux else out.cpu().numpy()


def oracle_dlnl(oracle, wl, odata, aux=False):
    return oracle.delta_loglike(oracle.Config(), odata, wl.params_new, wl.params_old, wl.walker_index,
                                move=wl.move, move_all=wl.move_all, N=wl.N, n_bins=wl.n_bins,
                                want_aux=aux, nthreads=oracle.max_threads())


# ------------------------------------------------------------------------------------------- waveform
@pytest.mark.parametrize("N", [128, 256, 512, 1024])
def test_waveform_each_window_length(oracle, torch_cuda, gb, N):
    """Several hundred sources over the whole 0.1-15 mHz range at one N: many CTAs, a ragged tail of the
    persistent loop (B not a multiple of the grid), every FFT plan."""
    gbfit, ctx = gb
    B = 1237
    p = make_workload(2, B=B).params_new
    ref, ref_k = oracle.waveform_batch(oracle.Config(), p, N=N, nthreads=oracle.max_threads())
    got, k = ctx.waveform(dev(torch_cuda, p), N=N)
    ctx.check()
    assert np.array_equal(k.cpu().numpy(), ref_k)
    e = wf_err(got.cpu().numpy(), ref)
    assert e <= TOL_WF, e


def test_waveform_mixed_n_bins_and_pitch(oracle, torch_cuda, gb):
    """Per-row N with a row pitch Nmax = 1024; elements beyond a row's N are left untouched."""
    gbfit, ctx = gb
    B = 777
    wl = make_workload(3, B=B, n_walkers=1)
    ref, ref_k = oracle.waveform_batch(oracle.Config(), wl.params_new, n_bins=wl.n_bins,
                                       nthreads=oracle.max_threads())
    sentinel = 7.0 - 3.0j
    out = torch_cuda.full((B, 2, 1024), sentinel, dtype=torch_cuda.complex128, device="cuda:0")
    got, k = ctx.waveform(dev(torch_cuda, wl.params_new), n_bins=dev(torch_cuda, wl.n_bins), Nmax=1024, out=out)
    ctx.check()
    got = got.cpu().numpy()
    assert np.array_equal(k.cpu().numpy(), ref_k)
    assert set(np.unique(wl.n_bins)) == {128, 256, 512, 1024}
    full = np.zeros((B, 2, 1024), np.complex128)
    full[:, :, :ref.shape[2]] = ref
    assert wf_err(got, full, wl.n_bins) <= TOL_WF
    for b in range(B):
        assert np.all(got[b, :, wl.n_bins[b]:] == sentinel)


def test_waveform_special_parameters(oracle, torch_cuda, gb):
    """Degenerate cases of the method: face-on, edge-on, ecliptic pole, delta = 0 and delta = +-1/2 (carrier
    exactly on / half-way between bins), fdot = 0, extreme fdot."""
    gbfit, ctx = gb
    T = 31457280.0
    base = np.array([2e-22, 3e-3, 1e-17, 0.4, 0.3, 0.9, 2.2, 0.35])
    rows = []
    for ci, sb in [(1.0, 0.2), (-1.0, -0.4), (0.0, 0.0), (0.4, 1.0), (0.4, -1.0), (0.0, 0.999999999)]:
        p = base.copy(); p[4], p[7] = ci, sb; rows.append(p)
    for q, frac in [(94372, 0.0), (94372, 0.5), (94373, -0.5), (31458, 0.25), (440000, 0.49999)]:
        p = base.copy(); p[1] = (q + frac) / T; rows.append(p)
    for fd in (0.0, 1e-16, -1e-16, 5e-15):
        p = base.copy(); p[2] = fd; p[1] = 12e-3; rows.append(p)
    p = np.array(rows)
    for N in (128, 1024):
        ref, ref_k = oracle.waveform_batch(oracle.Config(), p, N=N)
        got, k = ctx.waveform(dev(torch_cuda, p), N=N)
        ctx.check()
        assert np.array_equal(k.cpu().numpy(), ref_k)
        assert wf_err(got.cpu().numpy(), ref) <= TOL_WF


# --------------------------------------------------------------------------------- configs 1-4, full size
def test_config1_tiny_add_full(oracle, torch_cuda, gb):
    gbfit, ctx = gb
    wl = make_workload(1)
    resid = wl.resid()
    data, _ = upload(torch_cuda, gbfit, wl, resid)
    got, aux = gpu_dlnl(torch_cuda, gbfit, ctx, wl, data, aux=True)
    ref, raux = oracle_dlnl(oracle, wl, oracle.Data(resid, wl.psd, wl.k_lo), aux=True)
    assert np.abs(got - ref).max() <= TOL_DLNL
    assert np.abs(aux - raux).max() <= TOL_DLNL
    # windows that stick out of the 1-4 mHz band exist in this config (reading S13)
    q = np.floor(wl.params_new[:, 1] * wl.Tobs + 0.5)
    assert ((q - 64 < wl.k_lo) | (q + 64 > wl.k_lo + wl.n_f)).any()


def test_config2_add4096_full(oracle, torch_cuda, gb):
    gbfit, ctx = gb
    wl = make_workload(2)
    resid = wl.resid()
    data, _ = upload(torch_cuda, gbfit, wl, resid)
    got, aux = gpu_dlnl(torch_cuda, gbfit, ctx, wl, data, aux=True)
    ref, raux = oracle_dlnl(oracle, wl, oracle.Data(resid, wl.psd, wl.k_lo), aux=True)
    assert np.abs(got - ref).max() <= TOL_DLNL, np.abs(got - ref).max()
    assert np.abs(aux - raux).max() <= TOL_DLNL
    # and the waveforms of the same rows
    wref, kref = oracle.waveform_batch(oracle.Config(), wl.params_new, N=256, nthreads=oracle.max_threads())
    wgot, k = ctx.waveform(dev(torch_cuda, wl.params_new), N=256)
    assert np.array_equal(k.cpu().numpy(), kref)
    assert wf_err(wgot.cpu().numpy(), wref) <= TOL_WF


def test_config3_mixed_add_remove_full(oracle, torch_cuda, gb):
    gbfit, ctx = gb
    wl = make_workload(3)
    resid = wl.resid()
    data, _ = upload(torch_cuda, gbfit, wl, resid)
    got = gpu_dlnl(torch_cuda, gbfit, ctx, wl, data)
    ref = oracle_dlnl(oracle, wl, oracle.Data(resid, wl.psd, wl.k_lo))
    err = np.abs(got - ref)
    assert err.max() <= TOL_DLNL, (err.max(), int(err.argmax()))


def test_config4_swap_full(oracle, torch_cuda, gb):
    gbfit, ctx = gb
    wl = make_workload(4)
    resid = wl.resid()
    data, _ = upload(torch_cuda, gbfit, wl, resid)
    got = gpu_dlnl(torch_cuda, gbfit, ctx, wl, data)
    ref = oracle_dlnl(oracle, wl, oracle.Data(resid, wl.psd, wl.k_lo))
    err = np.abs(got - ref)
    assert err.max() <= TOL_DLNL, (err.max(), int(err.argmax()))
    # offset windows are exercised (q_new != q_old for a few per cent of the pairs)
    qn = np.floor(wl.params_new[:, 1] * wl.Tobs + 0.5)
    qo = np.floor(wl.params_old[:, 1] * wl.Tobs + 0.5)
    assert 0.005 < (qn != qo).mean() < 0.1


# ------------------------------------------------------------------------------ residual update (O9)
def test_residual_update_mixed_moves(oracle, torch_cuda, gb):
    """ADD / REMOVE / SWAP rows with an accepted mask, overlapping windows inside each walker: the atomic
    scatter equals the oracle's sequential update to rounding (sum order differs: reading S15)."""
    gbfit, ctx = gb
    B = 3000
    wl = make_workload(3, B=B, n_walkers=3)
    rng = np.random.Generator(np.random.Philox(key=[77, 1]))
    move = wl.move.copy()
    sw = rng.random(B) < 0.3
    move[sw] = 2
    pnew = wl.params_new.copy()
    pnew[sw, 1] += 1e-9 * rng.standard_normal(sw.sum())
    pnew[sw, 0] *= 1.02
    acc = (rng.random(B) < 0.5).astype(np.uint8)
    resid = wl.resid()
    data, d_resid = upload(torch_cuda, gbfit, wl, resid)
    ctx.residual_update(data, dev(torch_cuda, pnew), dev(torch_cuda, wl.params_old), dev(torch_cuda, wl.walker_index),
                        move=dev(torch_cuda, move), accepted=dev(torch_cuda, acc), n_bins=dev(torch_cuda, wl.n_bins))
    ctx.check()
    od = oracle.Data(resid.copy(), wl.psd, wl.k_lo)
    oracle.residual_update(oracle.Config(), od, pnew, wl.params_old, wl.walker_index, move=move, accepted=acc,
                           n_bins=wl.n_bins, nthreads=oracle.max_threads())
    got = d_resid.cpu().numpy()
    delta_ref = od.resid - resid
    delta_got = got - resid
    assert np.abs(delta_ref).max() > 0
    # compare the applied change (the noise floor is ~1e3 x larger than most waveforms)
    assert np.abs(delta_got - delta_ref).max() <= 1e-9 * np.abs(delta_ref).max()
    untouched = delta_ref == 0
    assert np.array_equal(got[untouched], resid[untouched])


def test_add_update_remove_roundtrip(oracle, torch_cuda, gb):
    """Invariant P6 on the GPU: after an accepted ADD is scattered, REMOVE of the same source has
    delta lnL = -(delta lnL of the ADD), and scattering the REMOVE restores the residual to rounding."""
    gbfit, ctx = gb
    wl = make_workload(2, B=1)
    p = wl.params_new.copy()
    p[0, 1] = 5.123456e-3
    wl.params_new = p
    resid = wl.resid()
    data, d_resid = upload(torch_cuda, gbfit, wl, resid)
    d_p, d_w = dev(torch_cuda, p), dev(torch_cuda, wl.walker_index)
    add = ctx.delta_loglike(data, d_p, None, d_w, move_all=gbfit.ADD, N=512).cpu().numpy()
    ctx.residual_update(data, d_p, None, d_w, move_all=gbfit.ADD, N=512)
    rem = ctx.delta_loglike(data, None, d_p, d_w, move_all=gbfit.REMOVE, N=512).cpu().numpy()
    ctx.residual_update(data, None, d_p, d_w, move_all=gbfit.REMOVE, N=512)
    ctx.check()
    assert abs(add[0] + rem[0]) <= 1e-9 * max(1.0, abs(add[0]))
    back = d_resid.cpu().numpy()
    # (r - a) + a differs from r by rounding at the scale of max(|r|, |a|)
    wf, _ = ctx.waveform(d_p, N=512)
    scale = max(np.abs(resid).max(), float(wf.abs().max()))
    assert np.abs(back - resid).max() <= 4e-16 * scale


def test_swap_identities(oracle, torch_cuda, gb):
    """swap(new = old) = 0 and swap = remove + add evaluated on the updated residual."""
    gbfit, ctx = gb
    wl = make_workload(4, B=64, n_walkers=2)
    resid = wl.resid()
    data, d_resid = upload(torch_cuda, gbfit, wl, resid)
    d_o, d_n, d_w = dev(torch_cuda, wl.params_old), dev(torch_cuda, wl.params_new), dev(torch_cuda, wl.walker_index)
    same = ctx.delta_loglike(data, d_o, d_o, d_w, move_all=gbfit.SWAP, N=512).cpu().numpy()
    assert np.abs(same).max() <= 1e-9
    sw = ctx.delta_loglike(data, d_n, d_o, d_w, move_all=gbfit.SWAP, N=512).cpu().numpy()
    # row by row: remove old, scatter, add new on the updated residual
    for b in range(8):
        sl = slice(b, b + 1)
        rem = ctx.delta_loglike(data, None, d_o[sl], d_w[sl], move_all=gbfit.REMOVE, N=512).cpu().numpy()[0]
        ctx.residual_update(data, None, d_o[sl], d_w[sl], move_all=gbfit.REMOVE, N=512)
        add = ctx.delta_loglike(data, d_n[sl], None, d_w[sl], move_all=gbfit.ADD, N=512).cpu().numpy()[0]
        ctx.residual_update(data, d_o[sl], None, d_w[sl], move_all=gbfit.ADD, N=512)   # put old back
        assert abs(sw[b] - (rem + add)) <= 1e-8 * max(1.0, abs(rem), abs(add)), (b, sw[b], rem, add)
    ctx.check()


# ---------------------------------------------------------------------------------- data-view options
def test_inverse_psd_and_walker_psd_map(oracle, torch_cuda, gb):
    gbfit, ctx = gb
    wl = make_workload(3, B=500, n_walkers=5)
    resid = wl.resid()
    wmap = np.array([2, 0, 1, 1, 0], np.int32)
    psd3 = wl.psd[:3]
    ref = oracle.delta_loglike(oracle.Config(), oracle.Data(resid, psd3, wl.k_lo, walker_psd=wmap),
                               wl.params_new, wl.params_old, wl.walker_index, move=wl.move, n_bins=wl.n_bins,
                               nthreads=oracle.max_threads())
    args = (dev(torch_cuda, wl.params_new), dev(torch_cuda, wl.params_old), dev(torch_cuda, wl.walker_index))
    kw = dict(move=dev(torch_cuda, wl.move), n_bins=dev(torch_cuda, wl.n_bins))
    d_resid = dev(torch_cuda, resid)
    d1 = gbfit.Data(d_resid, dev(torch_cuda, psd3), wl.k_lo, walker_psd=dev(torch_cuda, wmap))
    d2 = gbfit.Data(d_resid, dev(torch_cuda, 1.0 / psd3), wl.k_lo, walker_psd=dev(torch_cuda, wmap),
                    psd_is_inverse=True)
    g1 = ctx.delta_loglike(d1, *args, **kw).cpu().numpy()
    g2 = ctx.delta_loglike(d2, *args, **kw).cpu().numpy()
    ctx.check()
    assert np.abs(g1 - ref).max() <= TOL_DLNL
    assert np.abs(g2 - ref).max() <= TOL_DLNL


def test_host_forms_equal_device_forms(oracle, torch_cuda, gb):
    """The *_host entry points (pinned host buffers in and out) give the same bits as the device forms."""
    gbfit, ctx = gb
    torch = torch_cuda
    wl = make_workload(3, B=2000, n_walkers=4)
    resid = wl.resid()
    data, d_resid = upload(torch, gbfit, wl, resid)
    dl_dev = gpu_dlnl(torch, gbfit, ctx, wl, data)
    pin = lambda a: None if a is None else torch.as_tensor(np.ascontiguousarray(a)).pin_memory()
    out = torch.empty(wl.B, dtype=torch.float64).pin_memory()
    ctx.delta_loglike_host(data, pin(wl.params_new), pin(wl.params_old), pin(wl.walker_index), move=pin(wl.move),
                           n_bins=pin(wl.n_bins), out=out)
    assert np.array_equal(out.numpy(), dl_dev)
    wf_dev, k_dev = ctx.waveform(dev(torch, wl.params_new), n_bins=dev(torch, wl.n_bins), Nmax=1024)
    wf_h, k_h = ctx.waveform_host(wl.params_new, n_bins=wl.n_bins, Nmax=1024)
    assert np.array_equal(k_h, k_dev.cpu().numpy())
    assert np.array_equal(wf_h, wf_dev.cpu().numpy())
    acc = (np.arange(wl.B) % 4 == 0).astype(np.uint8)
    ctx.residual_update_host(data, wl.params_new, wl.params_old, wl.walker_index, move=wl.move, accepted=acc,
                             n_bins=wl.n_bins)
    od = oracle.Data(resid.copy(), wl.psd, wl.k_lo)
    oracle.residual_update(oracle.Config(), od, wl.params_new, wl.params_old, wl.walker_index, move=wl.move,
                           accepted=acc, n_bins=wl.n_bins, nthreads=oracle.max_threads())
    dref = od.resid - resid
    assert np.abs((d_resid.cpu().numpy() - resid) - dref).max() <= 1e-9 * np.abs(dref).max()


# ------------------------------------------------------------------------------------------ edge cases
def test_empty_batch_and_argument_errors(torch_cuda, gb):
    gbfit, ctx = gb
    torch = torch_cuda
    wl = make_workload(1, B=4)
    data, _ = upload(torch, gbfit, wl, wl.resid())
    empty_p = torch.empty((0, 8), dtype=torch.float64, device="cuda:0")
    empty_w = torch.empty((0,), dtype=torch.int32, device="cuda:0")
    assert ctx.delta_loglike(data, empty_p, None, empty_w, N=128).shape[0] == 0
    wf, k = ctx.waveform(empty_p, N=128)
    assert wf.shape[0] == 0
    with pytest.raises(gbfit.GbError) as ei:
        ctx.delta_loglike(data, dev(torch, wl.params_new), None, dev(torch, wl.walker_index), N=100)
    assert ei.value.code == gbfit.GB_ERR_INVALID
    with pytest.raises(gbfit.GbError):
        ctx.delta_loglike(data, None, None, dev(torch, wl.walker_index), N=128)   # ADD needs params_new
    with pytest.raises(gbfit.GbError):
        ctx.delta_loglike(data, dev(torch, wl.params_new), None, dev(torch, wl.walker_index), N=128, move_all=7)
    ctx.check()


def test_bad_rows_give_nan_and_sticky_flag(oracle, torch_cuda, gb):
    gbfit, ctx = gb
    torch = torch_cuda
    wl = make_workload(1, B=16)
    resid = wl.resid()
    data, _ = upload(torch, gbfit, wl, resid)
    w = wl.walker_index.copy(); w[3] = 5; w[7] = -1
    nb = np.full(16, 128, np.int32); nb[11] = 200
    out = ctx.delta_loglike(data, dev(torch, wl.params_new), None, dev(torch, w), n_bins=dev(torch, nb)).cpu().numpy()
    with pytest.raises(gbfit.GbError) as ei:
        ctx.check()
    assert ei.value.code == gbfit.GB_ERR_ROW
    ctx.check()                                     # the flag was cleared
    bad = np.zeros(16, bool); bad[[3, 7, 11]] = True
    assert np.isnan(out[bad]).all() and np.isfinite(out[~bad]).all()
    ref = oracle.delta_loglike(oracle.Config(), oracle.Data(resid, wl.psd, wl.k_lo), wl.params_new[~bad], None,
                               wl.walker_index[~bad], N=128)
    assert np.abs(out[~bad] - ref).max() <= TOL_DLNL


def test_window_fully_or_partly_outside_band(oracle, torch_cuda, gb):
    """Reading S13: bins outside [k_lo, k_lo + n_f) contribute nothing and are not scattered."""
    gbfit, ctx = gb
    torch = torch_cuda
    wl = make_workload(1, B=6)
    T = wl.Tobs
    p = wl.params_new.copy()
    p[:, 1] = [(wl.k_lo - 200) / T, (wl.k_lo - 10.3) / T, (wl.k_lo + 20.2) / T,
               (wl.k_lo + wl.n_f - 30.7) / T, (wl.k_lo + wl.n_f + 17.1) / T, (wl.k_lo + wl.n_f + 500) / T]
    resid = wl.resid()
    data, d_resid = upload(torch, gbfit, wl, resid)
    got = ctx.delta_loglike(data, dev(torch, p), None, dev(torch, wl.walker_index), N=128).cpu().numpy()
    od = oracle.Data(resid.copy(), wl.psd, wl.k_lo)
    ref = oracle.delta_loglike(oracle.Config(), od, p, None, wl.walker_index, N=128)
    assert got[0] == 0.0 and got[5] == 0.0
    assert np.abs(got - ref).max() <= TOL_DLNL
    ctx.residual_update(data, dev(torch, p), None, dev(torch, wl.walker_index), N=128)
    ctx.check()
    oracle.residual_update(oracle.Config(), od, p, None, wl.walker_index, N=128)
    dref = od.resid - resid
    assert np.abs((d_resid.cpu().numpy() - resid) - dref).max() <= 1e-9 * np.abs(dref).max()


def test_highest_bins_up_to_nyquist(oracle, torch_cuda, gb):
    """Maximum sizes: N = 1024 windows near the top of the stored band (30 mHz) and a window that would
    cross the Nyquist bin (rejected with the sticky flag)."""
    gbfit, ctx = gb
    torch = torch_cuda
    T = 31457280.0
    base = np.array([1e-22, 29.98e-3, 0.0, 1.0, 0.1, 0.2, 3.0, -0.3])
    ref, kref = oracle.waveform_batch(oracle.Config(), base[None, :], N=1024)
    got, k = ctx.waveform(dev(torch, base[None, :]), N=1024)
    ctx.check()
    assert np.array_equal(k.cpu().numpy(), kref)
    assert wf_err(got.cpu().numpy(), ref) <= TOL_WF
    p = base.copy(); p[1] = 0.1 - 100 / T          # Nyquist of dt = 5 s is 0.1 Hz
    ctx.waveform(dev(torch, p[None, :]), N=1024)
    with pytest.raises(gbfit.GbError):
        ctx.check()


# ----------------------------------------------------- fast / general slow-part dispatch (csrc/gb_fast.cuh)
def test_rows_inside_and_outside_the_fast_path_limits_in_one_batch(oracle, torch_cuda, gb):
    """gb_prep_kernel routes a row to the polynomial fast path or to the general kernels by its parameters
    (f0 > 30.5 mHz, |fdot| >~ 5e-13, |phi0| in the thousands, f0 <= 0 go the general way).  One batch with
    both kinds, mixed window lengths and all three moves must match the oracle row by row."""
    gbfit, ctx = gb
    torch = torch_cuda
    wl = make_workload(3, B=96, n_walkers=3)
    pn, po = wl.params_new.copy(), wl.params_old.copy()
    move = wl.move.copy()
    move[::4] = gbfit.SWAP
    pn[::4] = po[::4]
    pn[::4, 1] += 3e-9
    pn[::4, 3] += 0.02
    for arr in (pn, po):                # every 3rd row leaves the fast limits in one of three ways
        arr[1::6, 2] = 4e-12            # |fdot| beyond the first-order limit
        arr[2::6, 3] += 3500.0          # phase beyond the Cody-Waite range of the fast path
        arr[4::12, 1] = 4.2e-2          # above 30.5 mHz (window outside the stored band: delta lnL = 0)
    nb = wl.n_bins.copy()
    nb[4::12] = 1024
    resid = wl.resid()
    data, d_resid = upload(torch, gbfit, wl, resid)
    od = oracle.Data(resid.copy(), wl.psd, wl.k_lo, walker_psd=wl.walker_psd)
    ref = oracle.delta_loglike(oracle.Config(), od, pn, po, wl.walker_index, move=move, n_bins=nb,
                               nthreads=oracle.max_threads())
    got = ctx.delta_loglike(data, dev(torch, pn), dev(torch, po), dev(torch, wl.walker_index),
                            move=dev(torch, move), n_bins=dev(torch, nb)).cpu().numpy()
    ctx.check()
    assert np.abs(got - ref).max() <= TOL_DLNL
    refw, refk = oracle.waveform_batch(oracle.Config(), pn, n_bins=nb, nthreads=oracle.max_threads())
    gw, gk = ctx.waveform(dev(torch, pn), n_bins=dev(torch, nb), Nmax=int(refw.shape[2]))
    ctx.check()
    assert np.array_equal(gk.cpu().numpy(), refk)
    assert wf_err(gw.cpu().numpy(), refw, nb) <= TOL_WF
    acc = (np.arange(wl.B) % 2 == 0).astype(np.uint8)
    ctx.residual_update(data, dev(torch, pn), dev(torch, po), dev(torch, wl.walker_index), move=dev(torch, move),
                        accepted=dev(torch, acc), n_bins=dev(torch, nb))
    ctx.check()
    oracle.residual_update(oracle.Config(), od, pn, po, wl.walker_index, move=move, accepted=acc, n_bins=nb,
                           nthreads=oracle.max_threads())
    dref = od.resid - resid
    assert np.abs((d_resid.cpu().numpy() - resid) - dref).max() <= 1e-9 * np.abs(dref).max()


def test_sources_along_link_directions(oracle, torch_cuda, gb):
    """kappa -> +-1 at some time samples: the fast path's shared reciprocal is singular there and the sinc
    series takes over for that link (a degenerate case of the restructured arithmetic)."""
    gbfit, ctx = gb
    cfg = oracle.Config()
    rows = []
    for t in (0.0, 0.31 * cfg.Tobs, 0.77 * cfg.Tobs):
        x = oracle.orbits(cfg, float(t))
        for (r, s_), sign in (((0, 1), 1.0), ((2, 0), -1.0), ((1, 2), 1.0)):
            n = (x[r] - x[s_]) / cfg.armlength
            kdir = sign * n / np.linalg.norm(n)          # k = -(cos b cos l, cos b sin l, sin b)
            lam = np.arctan2(-kdir[1], -kdir[0]) % (2 * np.pi)
            for f0 in (2.5e-4, 2e-3, 1.2e-2):
                rows.append([1e-22, f0, 2e-17, 1.0, 0.3, 0.7, lam, -kdir[2]])
    p = np.array(rows)
    nb = n_bins_for_f0(p[:, 1])
    ref, refk = oracle.waveform_batch(cfg, p, n_bins=nb, nthreads=oracle.max_threads())
    got, k = ctx.waveform(dev(torch_cuda, p), n_bins=dev(torch_cuda, nb), Nmax=int(ref.shape[2]))
    ctx.check()
    assert np.array_equal(k.cpu().numpy(), refk)
    assert wf_err(got.cpu().numpy(), ref, nb) <= TOL_WF


# ------------------------------------------------------------------------ config 5: full-size launch
def test_config5_full_size_sampled(oracle, torch_cuda, gb):
    """The bench's launch configuration: 360 residuals (10.8 GB), 4.32 M ADD-type evaluations in one call,
    then the scatter of the accepted 25 %.  The oracle checks (a) delta lnL on a seeded sample of rows and
    (b) the final residuals of 4 walkers (all of their 12 000 rows, sequentially)."""
    gbfit, ctx = gb
    torch = torch_cuda
    free, total = torch.cuda.mem_get_info(0)
    if free < 20e9:
        pytest.skip("needs ~13 GB of free device memory")
    wl = make_workload(5)
    assert wl.B == 4_320_000 and wl.n_walkers == 360
    d_resid = torch.empty((wl.n_walkers, 2, wl.n_f), dtype=torch.complex128, device="cuda:0")
    check_walkers = [0, 37, 181, 359]
    keep = {}
    for w in range(wl.n_walkers):
        row = wl.resid_row(w)
        d_resid[w].copy_(torch.from_numpy(row))
        if w in check_walkers:
            keep[w] = row
    data = gbfit.Data(d_resid, dev(torch, wl.psd), wl.k_lo, walker_psd=dev(torch, wl.walker_psd))
    d_p, d_w, d_nb = dev(torch, wl.params_new), dev(torch, wl.walker_index), dev(torch, wl.n_bins)
    got = ctx.delta_loglike(data, d_p, None, d_w, move_all=gbfit.ADD, n_bins=d_nb)
    ctx.check()
    got = got.cpu().numpy()
    assert np.isfinite(got).all()
    # (a) sampled rows: all rows of the sample live on the 4 kept walkers
    rng = np.random.Generator(np.random.Philox(key=[5, 99]))
    per = wl.B // wl.n_walkers
    sample = np.concatenate([w * per + rng.choice(per, 600, replace=False) for w in check_walkers])
    sub = wl.subset(sample)
    small = np.stack([keep[w] for w in check_walkers])
    remap = {w: i for i, w in enumerate(check_walkers)}
    sub_w = np.array([remap[int(w)] for w in sub.walker_index], np.int32)
    sub_psd_map = np.array([wl.walker_psd[w] for w in check_walkers], np.int32)
    od = oracle.Data(small.copy(), wl.psd, wl.k_lo, walker_psd=sub_psd_map)
    ref = oracle.delta_loglike(oracle.Config(), od, sub.params_new, None, sub_w, n_bins=sub.n_bins,
                               nthreads=oracle.max_threads())
    err = np.abs(got[sample] - ref)
    assert err.max() <= TOL_DLNL, (err.max(), int(sample[err.argmax()]))
    # (b) scatter of the accepted rows
    ctx.residual_update(data, d_p, None, d_w, move_all=gbfit.ADD, accepted=dev(torch, wl.accepted), n_bins=d_nb)
    ctx.check()
    rows = np.concatenate([np.arange(w * per, (w + 1) * per) for w in check_walkers])
    sub = wl.subset(rows)
    sub_w = np.repeat(np.arange(len(check_walkers), dtype=np.int32), per)
    oracle.residual_update(oracle.Config(), od, sub.params_new, None, sub_w, accepted=sub.accepted,
                           n_bins=sub.n_bins, nthreads=oracle.max_threads())
    for i, w in enumerate(check_walkers):
        dref = od.resid[i] - keep[w]
        dgot = d_resid[w].cpu().numpy() - keep[w]
        assert np.abs(dref).max() > 0
        assert np.abs(dgot - dref).max() <= 1e-9 * np.abs(dref).max(), w
    # (c) the call bench.py times: the same step as ONE gb_delta_loglike_accept call (8 walker chunks, fused update).  The
    #     residuals go back first (REMOVE of the same rows: equal to the initial ones to rounding); the seeded flags enter as
    #     log u = -inf / +inf, so the decisions must reproduce them exactly
    ctx.residual_update(data, None, d_p, d_w, move_all=gbfit.REMOVE, accepted=dev(torch, wl.accepted), n_bins=d_nb)
    logu = np.where(wl.accepted != 0, -np.inf, np.inf)
    store_bins = int(1.15 * wl.n_bins[wl.accepted != 0].astype(np.int64).sum()) + 1024
    dl2, acc2 = ctx.delta_loglike_accept(data, d_p, None, d_w, dev(torch, logu), move_all=gbfit.ADD, n_bins=d_nb,
                                         store_bins=store_bins, apply=1)
    ctx.check()
    assert np.array_equal(acc2.cpu().numpy() != 0, wl.accepted != 0)
    dl2 = dl2.cpu().numpy()
    assert np.abs(dl2[sample] - ref).max() <= TOL_DLNL and np.abs(dl2 - got).max() <= 1e-6
    for i, w in enumerate(check_walkers):
        dref = od.resid[i] - keep[w]
        dgot = d_resid[w].cpu().numpy() - keep[w]
        assert np.abs(dgot - dref).max() <= 1e-9 * np.abs(dref).max(), w


# ------------------------------------------------------------------- row f4: normalised overlap of source pairs
def test_overlap_pairs_against_oracle(oracle, torch_cuda, gb):
    """gb_overlap on config-4-shaped pairs (jittered copies, some with offset windows), mixed window lengths,
    several PSD rows, S_n and 1/S_n layouts, a zero-amplitude row and a row outside the fast-path limits."""
    gbfit, ctx = gb
    torch = torch_cuda
    wl = make_workload(4, B=300, n_walkers=4)
    a, c = wl.params_new.copy(), wl.params_old.copy()
    a[:100, 1] = np.linspace(2e-4, 1.4e-2, 100)               # spread the first 100 over all window lengths
    c[:100] = a[:100]
    c[:100, 1] += 8e-9
    c[:100, 6] += 0.1
    c[100:110, 1] += 2.0 / wl.Tobs * np.arange(10)            # up to 18 bins apart
    a[120, 0] = 0.0
    a[121, 2] = c[121, 2] = 2e-12
    nb = n_bins_for_f0(a[:, 1])
    rows = (np.arange(300) % 4).astype(np.int32)
    data_o = oracle.Data(np.zeros((1, 2, wl.n_f), np.complex128), wl.psd, wl.k_lo)
    ref, raux = oracle.overlap(oracle.Config(), data_o, a, c, psd_row=rows, n_bins=nb, nthreads=oracle.max_threads())
    for psd, inv in ((wl.psd, False), (1.0 / wl.psd, True)):
        view = gbfit.Data.psd_only(dev(torch, psd), wl.k_lo, psd_is_inverse=inv)
        aux = torch.zeros((300, 2), dtype=torch.float64, device="cuda:0")
        got = ctx.overlap(view, dev(torch, a), dev(torch, c), psd_row=dev(torch, rows), n_bins=dev(torch, nb), aux=aux)
        ctx.check()
        got, aux = got.cpu().numpy(), aux.cpu().numpy()
        assert np.abs(got - ref).max() <= 1e-10
        assert np.abs(aux - raux).max() <= 1e-9 * raux.max() and np.abs(aux / np.maximum(raux, 1e-300) - 1)[raux > 0].max() <= 1e-9
    assert got[120] == 0.0 and abs(got[:100]).max() <= 1.0 + 1e-12
    same = ctx.overlap(view, dev(torch, c), dev(torch, c), N=512).cpu().numpy()     # psd_row = NULL -> row 0
    assert np.abs(same[100:] - 1.0).max() <= 1e-12
    bad = rows.copy(); bad[5] = 9
    out = ctx.overlap(view, dev(torch, a), dev(torch, c), psd_row=dev(torch, bad), n_bins=dev(torch, nb))
    with pytest.raises(gbfit.GbError):
        ctx.check()
    assert np.isnan(out.cpu().numpy()[5])


def test_repeated_calls_give_identical_bits(oracle, torch_cuda, gb):
    """No sanitizer on this pool: a race in the ticket / record / window pipeline or in the shared-memory FFT would
    show up as run-to-run differences.  delta lnL and waveforms have a fixed summation order, so repeated calls on the
    same inputs must agree bit for bit (the atomic scatter of gb_residual_update is the one order-dependent step)."""
    gbfit, ctx = gb
    torch = torch_cuda
    wl = make_workload(3, B=40000, n_walkers=6)
    mv = wl.move.copy()
    mv[::7] = gbfit.SWAP
    data, _ = upload(torch, gbfit, wl, wl.resid())
    args = (dev(torch, wl.params_new), dev(torch, wl.params_old), dev(torch, wl.walker_index))
    kw = dict(move=dev(torch, mv), n_bins=dev(torch, wl.n_bins))
    first = ctx.delta_loglike(data, *args, **kw).cpu().numpy()
    wf0, _ = ctx.waveform(args[0][:4096], n_bins=kw["n_bins"][:4096], Nmax=1024)
    wf0 = wf0.cpu().numpy()
    for _ in range(4):
        again = ctx.delta_loglike(data, *args, **kw).cpu().numpy()
        assert np.array_equal(again, first)
        wf, _ = ctx.waveform(args[0][:4096], n_bins=kw["n_bins"][:4096], Nmax=1024)
        assert np.array_equal(wf.cpu().numpy(), wf0)
    ctx.check()


def test_keep_and_update_kept_equal_the_two_call_form(oracle, torch_cuda, gb):
    """gb_delta_loglike_keep gives the bits of gb_delta_loglike; gb_residual_update_kept equals the oracle's update (and
    gb_residual_update) on the accepted rows, negate undoes it, and the kept state does not survive another call."""
    gbfit, ctx = gb
    torch = torch_cuda
    wl = make_workload(3, B=6000, n_walkers=4)
    wl.params_new[10, 1] = 4.1e-2                     # a general-path row (window outside the band)
    wl.n_bins[10] = 1024
    wl.params_old[10] = wl.params_new[10]
    resid = wl.resid()
    data, d_resid = upload(torch, gbfit, wl, resid)
    args = (dev(torch, wl.params_new), dev(torch, wl.params_old), dev(torch, wl.walker_index))
    kw = dict(move=dev(torch, wl.move), n_bins=dev(torch, wl.n_bins))
    plain = ctx.delta_loglike(data, *args, **kw).cpu().numpy()
    kept = ctx.delta_loglike_keep(data, *args, sum_n_bins=int(wl.n_bins.sum()), **kw).cpu().numpy()
    assert np.array_equal(plain, kept)
    acc = (np.random.Generator(np.random.Philox(key=[9, 9])).random(wl.B) < 0.3).astype(np.uint8)
    ctx.residual_update_kept(data, dev(torch, acc))
    ctx.check()
    od = oracle.Data(resid.copy(), wl.psd, wl.k_lo)
    oracle.residual_update(oracle.Config(), od, wl.params_new, wl.params_old, wl.walker_index, move=wl.move, accepted=acc,
                           n_bins=wl.n_bins, nthreads=oracle.max_threads())
    dref = od.resid - resid
    assert np.abs((d_resid.cpu().numpy() - resid) - dref).max() <= 1e-9 * np.abs(dref).max()
    ctx.residual_update_kept(data, dev(torch, acc), negate=True)
    assert np.abs(d_resid.cpu().numpy() - resid).max() <= 4e-16 * max(np.abs(resid).max(), np.abs(dref).max())
    ctx.delta_loglike(data, *args, **kw)              # any other batched call drops the kept state
    with pytest.raises(gbfit.GbError):
        ctx.residual_update_kept(data, dev(torch, acc))
    with pytest.raises(gbfit.GbError):                # too small a sum_n_bins: row-error flag
        ctx.delta_loglike_keep(data, *args, sum_n_bins=128 * wl.B, **kw)
        ctx.check()
    mv = wl.move.copy(); mv[3] = gbfit.SWAP
    ctx.delta_loglike_keep(data, *args, sum_n_bins=int(wl.n_bins.sum()), move=dev(torch, mv), n_bins=kw["n_bins"])
    with pytest.raises(gbfit.GbError):
        ctx.check()


def test_update_kept_after_an_undersized_keep_call_touches_nothing_out_of_range(oracle, torch_cuda, gb):
    """gb_delta_loglike_keep with too small a sum_n_bins skips the stores past the capacity and sets flag 4;
    a following gb_residual_update_kept must skip exactly those rows (and flag them) instead of adding stale scratch:
    the rows it does apply equal the oracle's update of those rows."""
    gbfit, ctx = gb
    torch = torch_cuda
    wl = make_workload(3, B=3000, n_walkers=3)
    resid = wl.resid()
    data, d_resid = upload(torch, gbfit, wl, resid)
    args = (dev(torch, wl.params_new), dev(torch, wl.params_old), dev(torch, wl.walker_index))
    kw = dict(move=dev(torch, wl.move), n_bins=dev(torch, wl.n_bins))
    # make the scratch hold a previous, larger call's windows: stale data lies beyond the small call's capacity
    ctx.delta_loglike_keep(data, *args, sum_n_bins=int(wl.n_bins.sum()), **kw)
    ctx.check()
    small = int(wl.n_bins.sum()) // 2
    assert small >= 128 * wl.B
    ctx.delta_loglike_keep(data, *args, sum_n_bins=small, **kw)
    ctx.residual_update_kept(data)
    with pytest.raises(gbfit.GbError) as ei:
        ctx.check()
    assert ei.value.code == gbfit.GB_ERR_ROW
    got = d_resid.cpu().numpy() - resid
    # the scratch is laid out class by class (N = 128 first), so the small windows fit and the large ones were skipped
    assert np.abs(got).max() > 0
    full = oracle.Data(resid.copy(), wl.psd, wl.k_lo)
    oracle.residual_update(oracle.Config(), full, wl.params_new, wl.params_old, wl.walker_index, move=wl.move,
                           n_bins=wl.n_bins, nthreads=oracle.max_threads())
    dfull = full.resid - resid
    assert np.abs(got - dfull).max() > 1e-3 * np.abs(dfull).max()          # some rows were skipped ...
    assert np.abs(got).max() <= np.abs(dfull).max() * 1.5                  # ... and nothing foreign was added
    # half of the window bins covers all N = 128 and N = 256 rows (f0 < 4 mHz) and none of the N = 1024 rows (> 10 mHz)
    lo = int(0.9e-3 * wl.Tobs) - wl.k_lo
    hi = int(10.2e-3 * wl.Tobs) - wl.k_lo
    assert np.abs(dfull[:, :, hi:]).max() > 0 and not got[:, :, hi:].any()
    assert np.abs(got[:, :, :lo] - dfull[:, :, :lo]).max() <= 1e-9 * np.abs(dfull[:, :, :lo]).max()
    # a gb_data with fewer walkers than the keep call saw: rows of the missing walkers are skipped and flagged
    ctx.delta_loglike_keep(data, *args, sum_n_bins=int(wl.n_bins.sum()), **kw)
    d2 = dev(torch, resid[:2])
    data2 = gbfit.Data(d2, dev(torch, wl.psd[:2]), wl.k_lo)
    ctx.residual_update_kept(data2)
    with pytest.raises(gbfit.GbError):
        ctx.check()
    sel = wl.walker_index < 2
    ref2 = oracle.Data(resid[:2].copy(), wl.psd[:2], wl.k_lo)
    oracle.residual_update(oracle.Config(), ref2, wl.params_new[sel], wl.params_old[sel], wl.walker_index[sel],
                           move=wl.move[sel], n_bins=wl.n_bins[sel], nthreads=oracle.max_threads())
    dref = ref2.resid - resid[:2]
    assert np.abs((d2.cpu().numpy() - resid[:2]) - dref).max() <= 1e-9 * np.abs(dref).max()


def test_row_errors_for_oversized_window_null_side_and_bad_psd_row(oracle, torch_cuda, gb):
    """a per-row N larger than the pitch of AE_out, a per-row move whose parameter side is NULL, and a
    walker_psd entry outside [0, n_psd) are row errors (flag 1, NaN / untouched row), not overruns or device faults."""
    gbfit, ctx = gb
    torch = torch_cuda
    wl = make_workload(3, B=12, n_walkers=2)
    nb = np.full(12, 128, np.int32); nb[5] = 512
    out = torch.full((12, 2, 256), 7.0, dtype=torch.complex128, device="cuda:0")
    ctx.waveform(dev(torch, wl.params_new), n_bins=dev(torch, nb), Nmax=256, out=out)
    with pytest.raises(gbfit.GbError) as ei:
        ctx.check()
    assert ei.value.code == gbfit.GB_ERR_ROW
    o = out.cpu().numpy()
    assert np.all(o[5] == 7.0)                                             # the bad row is left untouched
    assert np.all(o[:, :, 128:][np.arange(12) != 5] == 7.0)                # nothing past a row's own window
    ref, _ = oracle.waveform_batch(oracle.Config(), wl.params_new[:5], N=128)
    assert wf_err(o[:5, :, :128], ref) <= TOL_WF
    # per-row moves with params_old = NULL: the REMOVE rows are row errors, the ADD rows are computed
    resid = wl.resid()
    data, _ = upload(torch, gbfit, wl, resid)
    d = ctx.delta_loglike(data, dev(torch, wl.params_new), None, dev(torch, wl.walker_index), move=dev(torch, wl.move),
                          n_bins=dev(torch, wl.n_bins)).cpu().numpy()
    with pytest.raises(gbfit.GbError):
        ctx.check()
    assert (wl.move == 1).any() and (wl.move == 0).any()
    assert np.isnan(d[wl.move == 1]).all() and np.isfinite(d[wl.move == 0]).all()
    # walker_psd entry out of range
    wp = np.array([0, 9], np.int32)
    dataw = gbfit.Data(dev(torch, resid), dev(torch, wl.psd), wl.k_lo, walker_psd=dev(torch, wp))
    d = ctx.delta_loglike(dataw, dev(torch, wl.params_new), dev(torch, wl.params_old), dev(torch, wl.walker_index),
                          move=dev(torch, wl.move), n_bins=dev(torch, wl.n_bins)).cpu().numpy()
    with pytest.raises(gbfit.GbError):
        ctx.check()
    assert np.isnan(d[wl.walker_index == 1]).all() and np.isfinite(d[wl.walker_index == 0]).all()


def test_search_stage_geometry_single_residual_many_walkers_per_band(oracle, torch_cuda, gb):
    """App. G's batch shape: sub-bands x temperatures x walkers, one source per walker, f0 confined to
    its sub-band, every row against the SAME residual row -- consecutive rows read the same few hundred bins (the opposite
    of config 5, where neighbouring rows share a walker but not a frequency).  60 bands x 3 x 40 = 7200 rows, all four
    window lengths; every row against the oracle."""
    from gb_inputs import make_search_stage
    gbfit, ctx = gb
    torch = torch_cuda
    wl = make_search_stage(n_bands=60, n_temps=3, n_walkers=40)
    assert set(np.unique(wl.n_bins)) == {128, 256, 512, 1024}
    resid = wl.resid()
    ref, raux = oracle.delta_loglike(oracle.Config(), oracle.Data(resid, wl.psd, wl.k_lo), wl.params_new, None, wl.walker_index,
                                     n_bins=wl.n_bins, want_aux=True, nthreads=oracle.max_threads())
    data, _ = upload(torch, gbfit, wl, resid)
    aux = torch.zeros((wl.B, 2), dtype=torch.float64, device="cuda:0")
    got = ctx.delta_loglike(data, dev(torch, wl.params_new), None, dev(torch, wl.walker_index), move_all=gbfit.ADD,
                            n_bins=dev(torch, wl.n_bins), aux=aux)
    ctx.check()
    assert np.abs(got.cpu().numpy() - ref).max() <= TOL_DLNL
    assert np.abs(aux.cpu().numpy() - raux).max() <= 1e-6
    snr = np.sqrt(raux[:, 0])
    assert 2.0 < np.median(snr) < 60.0
