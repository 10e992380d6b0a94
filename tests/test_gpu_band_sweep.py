"""Parity of gb_band_sweep (Algorithm 1) with the CPU oracle on the
same seeded band tasks: accept / reject decisions and final parameters bit-exact (both sides decide
beta dlnL + logq >= logu in FP64), delta lnL <= 1e-6 absolute, final residuals <= 1e-9 of the largest change.
"""
import numpy as np
import pytest

from gb_inputs import make_band_tasks, make_workload

pytestmark = pytest.mark.gpu

TOL_DLNL = 1e-6


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


def dev(torch, a):
    return torch.as_tensor(np.ascontiguousarray(a)).to("cuda:0")


def run_gpu(torch, gbfit, ctx, wl, bt, resid, tasks=None, logu=None, psd=None, inverse=False):
    t = bt.tasks if tasks is None else tasks
    packed = gbfit.pack_band_tasks(**t)
    d_resid = dev(torch, resid)
    data = gbfit.Data(d_resid, dev(torch, wl.psd if psd is None else psd), wl.k_lo, psd_is_inverse=inverse)
    d_params = dev(torch, bt.params)
    acc, dl = ctx.band_sweep(data, dev(torch, packed.view(np.uint8)), bt.N, int(max(t["n_stage"].max(), 1)), d_params,
                             dev(torch, bt.prop_k), dev(torch, bt.prop_params), dev(torch, bt.prop_logq),
                             dev(torch, bt.prop_logu if logu is None else logu))
    ctx.check()
    return acc.cpu().numpy(), dl.cpu().numpy(), d_params.cpu().numpy(), d_resid.cpu().numpy()


def run_oracle(oracle, wl, bt, resid, tasks=None, logu=None):
    data = oracle.Data(resid.copy(), wl.psd, wl.k_lo)
    params = bt.params.copy()
    acc, dl = oracle.band_sweep(oracle.Config(), data, bt.tasks if tasks is None else tasks, bt.N, params, bt.prop_k,
                                bt.prop_params, bt.prop_logq, bt.prop_logu if logu is None else logu)
    return acc, dl, params, data.resid


def compare(got, ref, resid):
    acc, dl, params, r1 = got
    racc, rdl, rparams, rr1 = ref
    assert np.array_equal(acc, racc), int((acc != racc).sum())
    assert np.abs(dl - rdl).max() <= TOL_DLNL
    assert np.array_equal(params, rparams)
    change = np.abs(rr1 - resid).max()
    assert np.abs(r1 - rr1).max() <= 1e-9 * change + 4e-16 * np.abs(resid).max()


@pytest.mark.parametrize("N,f_lo,n_bands,amp", [(128, 5e-4, 6, 2e-22), (256, 2e-3, 6, 2e-22), (512, 6e-3, 4, 4e-23),
                                                 (1024, 1.2e-2, 3, 1e-23)])
def test_band_sweep_each_window_length(oracle, torch_cuda, gb, N, f_lo, n_bands, amp):
    gbfit, ctx = gb
    wl = make_workload(3, B=1, n_walkers=3)
    bt = make_band_tasks(wl, N, f_lo, n_bands, n_src=5, n_prop=14, amp_lo=0.1 * amp, amp_hi=amp)
    resid = wl.resid()
    ref = run_oracle(oracle, wl, bt, resid)
    assert 0 < ref[0].sum() < ref[0].size
    compare(run_gpu(torch_cuda, gbfit, ctx, wl, bt, resid), ref, resid)


def test_band_sweep_all_accepted_all_rejected_no_write_back_and_inverse_psd(oracle, torch_cuda, gb):
    gbfit, ctx = gb
    torch = torch_cuda
    wl = make_workload(3, B=1, n_walkers=2)
    bt = make_band_tasks(wl, 256, 2.5e-3, 5, n_src=4, n_prop=12, stream=1)
    resid = wl.resid()
    for logu in (np.full_like(bt.prop_logu, -np.inf), np.full_like(bt.prop_logu, np.inf)):
        compare(run_gpu(torch, gbfit, ctx, wl, bt, resid, logu=logu), run_oracle(oracle, wl, bt, resid, logu=logu), resid)
    t2 = dict(bt.tasks, write_back=np.zeros_like(bt.tasks["write_back"]))
    got = run_gpu(torch, gbfit, ctx, wl, bt, resid, tasks=t2)
    ref = run_oracle(oracle, wl, bt, resid, tasks=t2)
    assert np.array_equal(got[3], resid) and np.array_equal(ref[3], resid)
    assert np.array_equal(got[0], ref[0]) and np.array_equal(got[2], ref[2]) and np.abs(got[1] - ref[1]).max() <= TOL_DLNL
    got = run_gpu(torch, gbfit, ctx, wl, bt, resid, psd=1.0 / wl.psd, inverse=True)
    compare(got, run_oracle(oracle, wl, bt, resid), resid)


def test_band_sweep_edges_rj_amplitude_switch_and_bad_tasks(oracle, torch_cuda, gb):
    """Staged range partly outside the stored band, an empty task, n_prop = 0, the RJ amplitude switch of
    PAPER.md:564 (amp = 0 on one side), a proposal outside the fast-path limits, and invalid tasks."""
    gbfit, ctx = gb
    torch = torch_cuda
    wl = make_workload(1)                                   # band 1-4 mHz only (k_lo = 31458)
    bt = make_band_tasks(wl, 128, 1e-3, 4, n_src=3, n_prop=8, stream=2)
    t = {k: v.copy() for k, v in bt.tasks.items()}
    t["k_first"][0] = wl.k_lo - 200                          # staged bins below the stored band
    t["n_prop"][1] = 0                                       # a task with nothing to do
    bt.params[t["src_begin"][0]:t["src_begin"][0] + 3, 1] = (wl.k_lo + 20 + np.arange(3) * 30) / wl.Tobs
    bt.prop_params[0:8, 1] = bt.params[t["src_begin"][0] + bt.prop_k[0:8], 1] + 1e-9
    p2 = t["prop_begin"][2]
    bt.prop_params[p2] = bt.params[t["src_begin"][2] + bt.prop_k[p2]]
    bt.prop_params[p2, 0] = 0.0                              # proposed removal: amplitude -> 0
    bt.prop_params[p2 + 1, 2] = 3e-12                        # outside the fast-path limits: general kernels' arithmetic
    resid = wl.resid()
    compare(run_gpu(torch, gbfit, ctx, wl, bt, resid, tasks=t), run_oracle(oracle, wl, bt, resid, tasks=t), resid)
    # invalid: walker out of range -> sticky flag, NaN rows
    bad = {k: v.copy() for k, v in bt.tasks.items()}
    bad["walker"][0] = 7
    packed = gbfit.pack_band_tasks(**bad)
    data = gbfit.Data(dev(torch, resid), dev(torch, wl.psd), wl.k_lo)
    acc, dl = ctx.band_sweep(data, dev(torch, packed.view(np.uint8)), 128, 384, dev(torch, bt.params), dev(torch, bt.prop_k),
                             dev(torch, bt.prop_params), dev(torch, bt.prop_logq), dev(torch, bt.prop_logu))
    with pytest.raises(gbfit.GbError):
        ctx.check()
    assert np.isnan(dl.cpu().numpy()[:8]).all() and np.isfinite(dl.cpu().numpy()[8:]).all()
    with pytest.raises(gbfit.GbError):
        ctx.band_sweep(data, dev(torch, packed.view(np.uint8)), 128, gbfit.BAND_MAX_STAGE + 1, dev(torch, bt.params),
                       dev(torch, bt.prop_k), dev(torch, bt.prop_params), dev(torch, bt.prop_logq), dev(torch, bt.prop_logu))


def test_band_sweep_odd_even_cold_chain_buffers(oracle, torch_cuda, gb):
    """Row f3 (Fig. 4): tasks stage from the EVEN buffer of their walker, subtract the band's current
    sources on chip, and the cold chain writes its accepted changes into the ODD buffer; hot chains store nothing."""
    from oddeven_setup import oddeven_case
    gbfit, ctx = gb
    torch = torch_cuda
    for N, f_lo, amp in ((128, 6e-4, 2e-22), (512, 6e-3, 4e-23)):
        wl, d, buf, wpsd, cold, tcold, hot, thot, ev = oddeven_case(oracle, N=N, f_lo=f_lo, n_bands=4, n_src=4, n_prop=12,
                                                                  n_walkers=3, amp=(0.1 * amp, amp))
        for bt, tt in ((cold, tcold), (hot, thot)):
            r_ref = buf.copy()
            p_ref = bt.params.copy()
            racc, rdl = oracle.band_sweep(oracle.Config(), oracle.Data(r_ref, wl.psd, wl.k_lo, walker_psd=wpsd), tt, N, p_ref,
                                          bt.prop_k, bt.prop_params, bt.prop_logq, bt.prop_logu)
            d_resid = dev(torch, buf)
            data = gbfit.Data(d_resid, dev(torch, wl.psd), wl.k_lo, walker_psd=dev(torch, wpsd))
            d_params = dev(torch, bt.params)
            acc, dl = ctx.band_sweep(data, dev(torch, gbfit.pack_band_tasks(**tt).view(np.uint8)), N, 3 * N, d_params,
                                     dev(torch, bt.prop_k), dev(torch, bt.prop_params), dev(torch, bt.prop_logq),
                                     dev(torch, bt.prop_logu))
            ctx.check()
            assert 0 < racc.sum() < racc.size
            compare((acc.cpu().numpy(), dl.cpu().numpy(), d_params.cpu().numpy(), d_resid.cpu().numpy()),
                    (racc, rdl, p_ref, r_ref), buf if tt["write_back"].any() else buf + 1e-30)
            assert np.array_equal(d_resid.cpu().numpy()[0::2], buf[0::2])     # even buffers are only read


def test_band_sweep_many_tasks_sampled(oracle, torch_cuda, gb):
    """The bench's launch shape at a tenth of its size: 36 walkers x 183 odd 256-bin sub-bands (6588 concurrent tasks,
    more than one wave of CTAs), 9 sources and 30 proposals each.  Tasks of one walker only share bins that none of their
    windows reach, and tasks of different walkers share nothing, so the oracle can run ALL 183 tasks of each of three
    walkers (549 tasks, in task order) on the initial residual: decisions, delta lnL and final parameters of those tasks
    and the walkers' whole written-back residual rows -- the place where concurrent CTAs add to one row with atomics --
    must match.  The other tasks are checked for finite output only."""
    gbfit, ctx = gb
    torch = torch_cuda
    wl = make_workload(3, B=1, n_walkers=36)
    bt = make_band_tasks(wl, 256, 1e-3, n_bands=183, n_src=9, n_prop=30)
    resid = wl.resid()
    d_resid = dev(torch, resid)
    data = gbfit.Data(d_resid, dev(torch, wl.psd), wl.k_lo)
    d_params = dev(torch, bt.params)
    acc, dl = ctx.band_sweep(data, dev(torch, gbfit.pack_band_tasks(**bt.tasks).view(np.uint8)), 256, bt.max_stage, d_params,
                             dev(torch, bt.prop_k), dev(torch, bt.prop_params), dev(torch, bt.prop_logq), dev(torch, bt.prop_logu))
    ctx.check()
    acc, dl, params = acc.cpu().numpy(), dl.cpu().numpy(), d_params.cpu().numpy()
    r1 = d_resid.cpu().numpy()
    nt = len(bt.tasks["walker"])
    assert nt == 6588 and np.isfinite(dl).all()
    walkers = (0, 17, 35)
    pick = np.flatnonzero(np.isin(bt.tasks["walker"], walkers))
    assert pick.size == 3 * 183
    sub = {k: v[pick] for k, v in bt.tasks.items()}
    p_ref = bt.params.copy()
    odata = oracle.Data(resid.copy(), wl.psd, wl.k_lo)
    racc, rdl = oracle.band_sweep(oracle.Config(), odata, sub, 256, p_ref, bt.prop_k, bt.prop_params, bt.prop_logq, bt.prop_logu)
    for i in pick:
        ps = slice(bt.tasks["prop_begin"][i], bt.tasks["prop_begin"][i] + bt.tasks["n_prop"][i])
        ss = slice(bt.tasks["src_begin"][i], bt.tasks["src_begin"][i] + bt.tasks["n_src"][i])
        assert np.array_equal(acc[ps], racc[ps]), i
        assert np.abs(dl[ps] - rdl[ps]).max() <= TOL_DLNL, i
        assert np.array_equal(params[ss], p_ref[ss]), i
    for w in walkers:                                   # the whole row: every task of the walker wrote into it
        change = np.abs(odata.resid[w] - resid[w]).max()
        assert change > 0
        assert np.abs(r1[w] - odata.resid[w]).max() <= 1e-9 * change + 4e-16 * np.abs(resid[w]).max(), w
    assert 0.02 < acc.mean() < 0.98


# ---------------------------------------------------------------------------------------------------------------------
# gb_band_sweep_generate: the proposal step of Algorithm 1 inside the kernel (App. B, Eq. 14)
def _stretch_pair(oracle, gbfit, torch, si, **over):
    f = dict(seed=si.seed, sweep=si.sweep, group=si.group, n_friends=si.n_friends, lo=si.lo, hi=si.hi, periodic=si.periodic,
             stretch_a=si.stretch_a)
    f.update(over)
    so = oracle.Stretch(f["seed"], f["sweep"], f["group"], f["n_friends"], f["lo"], f["hi"], f["periodic"], f["stretch_a"])
    sg = gbfit.Stretch(f["seed"], f["sweep"], dev(torch, f["group"]), f["n_friends"], f["lo"], f["hi"], f["periodic"],
                       f["stretch_a"])
    return so, sg


def _run_generate(oracle, torch, gbfit, ctx, wl, bt, resid, so, sg, tasks=None):
    t = bt.tasks if tasks is None else tasks
    odata = oracle.Data(resid.copy(), wl.psd, wl.k_lo)
    p_ref = bt.params.copy()
    ref = oracle.band_sweep_generate(oracle.Config(), odata, t, bt.N, p_ref, so)
    d_resid = dev(torch, resid)
    data = gbfit.Data(d_resid, dev(torch, wl.psd), wl.k_lo)
    d_params = dev(torch, bt.params)
    P = int((t["prop_begin"] + t["n_prop"]).max())
    got = ctx.band_sweep_generate(data, dev(torch, gbfit.pack_band_tasks(**t).view(np.uint8)), bt.N,
                                  int(max(t["n_stage"].max(), 1)), d_params, sg, P)
    ctx.check()
    got = [x.cpu().numpy() for x in got]
    return got, d_params.cpu().numpy(), d_resid.cpu().numpy(), ref, p_ref, odata.resid


def _compare_generate(got, params, r1, ref, p_ref, rr1, resid, rows=None):
    acc, dl, k, pp, lq, lu = got
    racc, rdl, rk, rpp, rlq, rlu = ref
    sl = slice(None) if rows is None else rows
    assert np.array_equal(k[sl], rk[sl])                               # randint: bit-exact
    assert np.array_equal(pp[sl], rpp[sl])                             # theta' (friend, z, Eq. 14, wrap): bit-exact
    assert np.abs(lq[sl] - rlq[sl]).max() <= 4e-15 and np.abs(lu[sl] - rlu[sl]).max() <= 2e-14   # libm log vs CUDA log
    assert np.array_equal(acc[sl], racc[sl]), int((acc[sl] != racc[sl]).sum())
    assert np.array_equal(np.isnan(dl[sl]), np.isnan(rdl[sl]))
    ok = np.isfinite(rdl[sl])
    assert np.abs(dl[sl][ok] - rdl[sl][ok]).max() <= TOL_DLNL
    if rows is None:
        assert np.array_equal(params, p_ref)
        change = np.abs(rr1 - resid).max()
        assert np.abs(r1 - rr1).max() <= 1e-9 * change + 4e-16 * np.abs(resid).max()


@pytest.mark.parametrize("N,f_lo,n_bands,amp", [(128, 5e-4, 6, 2e-22), (256, 2e-3, 6, 2e-22), (512, 6e-3, 4, 4e-23),
                                                 (1024, 1.2e-2, 3, 1e-23)])
def test_band_sweep_generate_each_window_length(oracle, torch_cuda, gb, N, f_lo, n_bands, amp):
    """k and theta' bit-exact, decisions equal, delta lnL <= 1e-6, final parameters bit-exact, residuals <= 1e-9 of the
    change (tasks of one walker have disjoint stages -- band_stride = 4 -- and proposals are confined to the stage, so the
    order in which tasks run does not matter); the case contains a source that is proposed again after an accepted proposal (so theta' was built from the
    NEW theta_k: a caller-side pre-generated proposal could not reproduce it)."""
    from gb_inputs import make_stretch_inputs
    gbfit, ctx = gb
    wl = make_workload(3, B=1, n_walkers=3)
    bt = make_band_tasks(wl, N, f_lo, n_bands, n_src=4, n_prop=16, amp_lo=0.1 * amp, amp_hi=amp, band_stride=4)
    si = make_stretch_inputs(bt, n_copies=6, n_friends=8)
    so, sg = _stretch_pair(oracle, gbfit, torch_cuda, si)
    resid = wl.resid()
    got, params, r1, ref, p_ref, rr1 = _run_generate(oracle, torch_cuda, gbfit, ctx, wl, bt, resid, so, sg)
    racc, rk = ref[0], ref[2]
    assert 0 < racc.sum() < racc.size
    again = 0
    t = bt.tasks
    for i in range(len(t["walker"])):
        moved = set()
        for p in range(t["n_prop"][i]):
            ip = t["prop_begin"][i] + p
            again += rk[ip] in moved
            if racc[ip]:
                moved.add(rk[ip])
    assert again > 0
    _compare_generate(got, params, r1, ref, p_ref, rr1, resid)


def test_band_sweep_generate_prior_box_wrap_small_group_and_errors(oracle, torch_cuda, gb):
    """Proposals outside a tight prior box (NaN, rejected, no evaluation), periodic wrap, a friends table smaller than
    n_friends, ties in f0, odd/even flags off / write_back off, and argument errors."""
    from gb_inputs import make_stretch_inputs
    gbfit, ctx = gb
    torch = torch_cuda
    wl = make_workload(3, B=1, n_walkers=2)
    bt = make_band_tasks(wl, 256, 2.5e-3, 5, n_src=3, n_prop=12, stream=3, band_stride=4)
    resid = wl.resid()
    si = make_stretch_inputs(bt, n_copies=4, n_friends=6, scale=8.0)          # wide group: wraps and box exits happen
    lo, hi = si.lo.copy(), si.hi.copy()
    lo[0], hi[0] = 3e-23, 1.5e-22                                             # tight amplitude prior
    so, sg = _stretch_pair(oracle, gbfit, torch, si, lo=lo, hi=hi)
    got, params, r1, ref, p_ref, rr1 = _run_generate(oracle, torch, gbfit, ctx, wl, bt, resid, so, sg)
    assert 0 < np.isnan(ref[1]).sum() < ref[1].size
    raw = si.group[:, 3].min() < 0.3 and si.group[:, 3].max() > 5.9             # phases near both ends: wraps occur
    assert raw
    _compare_generate(got, params, r1, ref, p_ref, rr1, resid)
    # table smaller than n_friends, with equal f0 values
    grp = si.group[:5].copy()
    grp[1, 1] = grp[2, 1]
    so, sg = _stretch_pair(oracle, gbfit, torch, si, group=grp, n_friends=9)
    t2 = dict(bt.tasks, write_back=np.zeros_like(bt.tasks["write_back"]))
    got, params, r1, ref, p_ref, rr1 = _run_generate(oracle, torch, gbfit, ctx, wl, bt, resid, so, sg, tasks=t2)
    assert np.array_equal(r1, resid)
    _compare_generate(got, params, r1, ref, p_ref, rr1, resid + 0.0)
    # errors: NULL table / a <= 1 are refused at the call; a task without sources is a row error
    with pytest.raises(gbfit.GbError):
        _run_generate(oracle, torch, gbfit, ctx, wl, bt, resid, so,
                      gbfit.Stretch(1, 1, dev(torch, grp), 4, si.lo, si.hi, si.periodic, stretch_a=1.0))
    bad = {k: v.copy() for k, v in bt.tasks.items()}
    bad["n_src"][0] = 0
    data = gbfit.Data(dev(torch, resid), dev(torch, wl.psd), wl.k_lo)
    out = ctx.band_sweep_generate(data, dev(torch, gbfit.pack_band_tasks(**bad).view(np.uint8)), 256, 768,
                                  dev(torch, bt.params), sg, bt.prop_k.size)
    with pytest.raises(gbfit.GbError):
        ctx.check()
    assert np.isnan(out[1].cpu().numpy()[:12]).all()


def test_band_sweep_generate_many_tasks_whole_walkers(oracle, torch_cuda, gb):
    """Launch scale (6588 tasks, more than one wave of CTAs) with a 0.7 M-row friends table: the oracle replays ALL tasks
    of three walkers; k, theta', decisions, parameters of those tasks and the walkers' written-back residual rows match."""
    from gb_inputs import make_stretch_inputs
    gbfit, ctx = gb
    torch = torch_cuda
    wl = make_workload(3, B=1, n_walkers=36)
    bt = make_band_tasks(wl, 256, 1e-3, n_bands=183, n_src=9, n_prop=30, band_stride=4)   # disjoint stages per walker
    si = make_stretch_inputs(bt, n_copies=12, n_friends=24)
    assert si.group.shape[0] == 36 * 183 * 9 * 12
    so, sg = _stretch_pair(oracle, gbfit, torch, si)
    resid = wl.resid()
    d_resid = dev(torch, resid)
    data = gbfit.Data(d_resid, dev(torch, wl.psd), wl.k_lo)
    d_params = dev(torch, bt.params)
    got = ctx.band_sweep_generate(data, dev(torch, gbfit.pack_band_tasks(**bt.tasks).view(np.uint8)), 256, bt.max_stage,
                                  d_params, sg, bt.prop_k.size)
    ctx.check()
    got = [x.cpu().numpy() for x in got]
    params, r1 = d_params.cpu().numpy(), d_resid.cpu().numpy()
    walkers = (0, 17, 35)
    pick = np.flatnonzero(np.isin(bt.tasks["walker"], walkers))
    sub = {k: v[pick] for k, v in bt.tasks.items()}
    p_ref = bt.params.copy()
    odata = oracle.Data(resid.copy(), wl.psd, wl.k_lo)
    ref = oracle.band_sweep_generate(oracle.Config(), odata, sub, 256, p_ref, so)
    for i in pick:
        ps = slice(bt.tasks["prop_begin"][i], bt.tasks["prop_begin"][i] + bt.tasks["n_prop"][i])
        ss = slice(bt.tasks["src_begin"][i], bt.tasks["src_begin"][i] + bt.tasks["n_src"][i])
        _compare_generate(got, None, None, ref, None, None, None, rows=ps)
        assert np.array_equal(params[ss], p_ref[ss]), i
    for w in walkers:
        change = np.abs(odata.resid[w] - resid[w]).max()
        assert change > 0
        assert np.abs(r1[w] - odata.resid[w]).max() <= 1e-9 * change + 4e-16 * np.abs(resid[w]).max(), w
    assert 0.02 < got[0].mean() < 0.98
