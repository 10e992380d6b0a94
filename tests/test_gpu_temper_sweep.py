"""Parity of gb_temper_sweep (Algorithm 2 with Eq. D2) with the CPU
oracle on the same seeded ladders: decisions and final permutations bit-exact, (D_i, D_j) <= 1e-6 absolute, final
residuals <= 1e-9 of the largest change."""
import numpy as np
import pytest

from temper_setup import temper_case

pytestmark = pytest.mark.gpu


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


def run_both(oracle, torch, gbfit, ctx, wl, tt, resid, tasks=None, logu=None, psd=None, inverse=False):
    t = tt.tasks if tasks is None else tasks
    lu = tt.chain_logu if logu is None else logu
    r_ref = resid.copy()
    ref = oracle.temper_sweep(oracle.Config(), oracle.Data(r_ref, wl.psd, wl.k_lo), t, tt.N, tt.params, tt.chain_walker,
                              tt.chain_beta, tt.chain_set_begin, tt.chain_set_n, lu)
    d_resid = dev(torch, resid)
    data = gbfit.Data(d_resid, dev(torch, wl.psd if psd is None else psd), wl.k_lo, psd_is_inverse=inverse)
    packed = gbfit.pack_temper_tasks(**t)
    got = ctx.temper_sweep(data, dev(torch, packed.view(np.uint8)), tt.N, int(t["n_stage"].max()), dev(torch, tt.params),
                           dev(torch, tt.chain_walker), dev(torch, tt.chain_beta), dev(torch, tt.chain_set_begin),
                           dev(torch, tt.chain_set_n), dev(torch, lu))
    ctx.check()
    perm, acc, dl = (x.cpu().numpy() for x in got)
    assert np.array_equal(acc, ref[1]), int((acc != ref[1]).sum())
    assert np.array_equal(perm, ref[0])
    assert np.abs(dl - ref[2]).max() <= 1e-6
    change = np.abs(r_ref - resid).max()
    assert np.abs(d_resid.cpu().numpy() - r_ref).max() <= 1e-9 * change + 4e-16 * np.abs(resid).max()
    return ref


@pytest.mark.parametrize("N,f_lo,amp", [(128, 6e-4, 2e-22), (256, 2e-3, 1e-22), (512, 6e-3, 3e-23), (1024, 1.2e-2, 8e-24)])
def test_temper_sweep_each_window_length(oracle, torch_cuda, gb, N, f_lo, amp):
    gbfit, ctx = gb
    wl, tt, resid = temper_case(oracle, N=N, f_lo=f_lo, n_bands=3, n_t=5, n_src=3, n_walkers=6, amp=(0.1 * amp, amp))
    ref = run_both(oracle, torch_cuda, gbfit, ctx, wl, tt, resid)
    assert ref[1].any()


def test_temper_sweep_all_accepted_none_accepted_no_write_back_inverse_psd_and_bad_tasks(oracle, torch_cuda, gb):
    gbfit, ctx = gb
    torch = torch_cuda
    wl, tt, resid = temper_case(oracle, N=256, f_lo=2.5e-3, n_bands=4, n_t=6, n_src=2, n_walkers=7, stream=3)
    for lu in (np.full_like(tt.chain_logu, -np.inf), np.full_like(tt.chain_logu, np.inf)):
        run_both(oracle, torch, gbfit, ctx, wl, tt, resid, logu=lu)
    t0 = dict(tt.tasks, write_back=np.zeros_like(tt.tasks["write_back"]))
    run_both(oracle, torch, gbfit, ctx, wl, tt, resid, tasks=t0, logu=np.full_like(tt.chain_logu, -np.inf))
    run_both(oracle, torch, gbfit, ctx, wl, tt, resid, psd=1.0 / wl.psd, inverse=True)
    # staged range partly below the stored band, a ladder of one chain (nothing to do), an empty set
    t1 = {k: v.copy() for k, v in tt.tasks.items()}
    t1["k_first"][0] = wl.k_lo - 5 * tt.N
    t1["n_t"][1] = 1
    sn = tt.chain_set_n.copy()
    sn[t1["chain_begin"][2] + 1] = 0
    import copy
    tt2 = copy.copy(tt)
    tt2.chain_set_n = sn
    run_both(oracle, torch, gbfit, ctx, wl, tt2, resid, tasks=t1)
    # invalid walker -> sticky flag and NaN for that ladder
    bad = tt.chain_walker.copy()
    bad[tt.tasks["chain_begin"][1] + 2] = 99
    data = gbfit.Data(dev(torch, resid), dev(torch, wl.psd), wl.k_lo)
    packed = gbfit.pack_temper_tasks(**tt.tasks)
    perm, acc, dl = ctx.temper_sweep(data, dev(torch, packed.view(np.uint8)), tt.N, tt.max_stage, dev(torch, tt.params),
                                     dev(torch, bad), dev(torch, tt.chain_beta), dev(torch, tt.chain_set_begin),
                                     dev(torch, tt.chain_set_n), dev(torch, tt.chain_logu))
    with pytest.raises(gbfit.GbError):
        ctx.check()
    cb = tt.tasks["chain_begin"][1]
    assert np.isnan(dl.cpu().numpy()[cb + 1:cb + 6]).all() and np.isfinite(dl.cpu().numpy()[:cb]).all()


def test_temper_sweep_many_ladders_sampled(oracle, torch_cuda, gb):
    """The bench's launch shape at reduced size: 183 odd 256-bin sub-bands x 4 disjoint walker groups = 732 ladders of
    8 chains running concurrently.  Ladders of one sub-band use disjoint residual rows and ladders of different
    sub-bands only share bins that no window of either reaches, so the oracle can run, on the initial residuals, every
    ladder that touches one of two chosen residual rows (2 x 183 ladders, one per sub-band each): decisions, (D_i, D_j)
    and permutations of those ladders and the two rows' whole written-back residuals must match."""
    gbfit, ctx = gb
    torch = torch_cuda
    from gb_inputs import make_workload, make_temper_tasks
    wl = make_workload(3, B=1, n_walkers=32)
    tt = make_temper_tasks(wl, 256, 1e-3, n_bands=183, n_t=8, n_src=6, n_groups=4)
    lu = tt.chain_logu.copy()
    lu[np.random.Generator(np.random.Philox(key=[2, 256])).random(lu.size) < 0.3] = -np.inf      # some accepted exchanges
    resid = wl.resid()
    d_resid = dev(torch, resid)
    data = gbfit.Data(d_resid, dev(torch, wl.psd), wl.k_lo)
    packed = gbfit.pack_temper_tasks(**tt.tasks)
    perm, acc, dl = ctx.temper_sweep(data, dev(torch, packed.view(np.uint8)), 256, tt.max_stage, dev(torch, tt.params),
                                     dev(torch, tt.chain_walker), dev(torch, tt.chain_beta), dev(torch, tt.chain_set_begin),
                                     dev(torch, tt.chain_set_n), dev(torch, lu))
    ctx.check()
    perm, acc, dl = perm.cpu().numpy(), acc.cpu().numpy(), dl.cpu().numpy()
    r1 = d_resid.cpu().numpy()
    nt = len(tt.tasks["n_t"])
    assert nt == 732 and np.isfinite(dl).all()
    rows = (3, 20)
    cw = tt.chain_walker.reshape(nt, 8)
    pick = np.flatnonzero(np.isin(cw, rows).any(axis=1))
    assert 183 <= pick.size <= 2 * 183 and all((cw == w).any(axis=1).sum() == 183 for w in rows)
    sub = {k: v[pick] for k, v in tt.tasks.items()}
    odata = oracle.Data(resid.copy(), wl.psd, wl.k_lo)
    rperm, racc, rdl = oracle.temper_sweep(oracle.Config(), odata, sub, 256, tt.params, tt.chain_walker, tt.chain_beta,
                                           tt.chain_set_begin, tt.chain_set_n, lu)
    for i in pick:
        cs = slice(tt.tasks["chain_begin"][i], tt.tasks["chain_begin"][i] + tt.tasks["n_t"][i])
        assert np.array_equal(acc[cs], racc[cs]) and np.array_equal(perm[cs], rperm[cs]), i
        assert np.abs(dl[cs] - rdl[cs]).max() <= 1e-6, i
    for w in rows:                                      # every ladder that writes into these rows was replayed
        change = np.abs(odata.resid[w] - resid[w]).max()
        assert change > 0
        assert np.abs(r1[w] - odata.resid[w]).max() <= 1e-9 * change + 4e-16 * np.abs(resid[w]).max(), w
    assert acc.sum() > 0


@pytest.mark.parametrize("N,f_lo,amp", [(128, 6e-4, 2e-22), (512, 6e-3, 3e-23)])
def test_temper_sweep_odd_even_cold_chain_buffers(oracle, torch_cuda, gb, N, f_lo, amp):
    """Row f2 on the data model of row f3 (Algorithm 2 as printed; buffers PAPER.md:354-362): ladders stage
    from rows that hold none of the band's sources, every chain's residual is formed on chip as row - (set it holds), and
    only exchanges with the cold chain are written, into the cold chain's own-parity row.  Decisions, permutations bit-exact,
    (D_i, D_j) <= 1e-6, written rows <= 1e-9 of the change, the staged-from rows untouched; a 24-chain ladder (the paper's
    temperature count) and a 33-chain one (beyond GB_TEMPER_MAX_LADDER_ODD_EVEN: row error)."""
    gbfit, ctx = gb
    torch = torch_cuda
    for n_t, n_walkers, n_groups in ((4, 12, 3), (24, 24, 1)):
        wl, tt, resid, d_rows = temper_case(oracle, N=N, f_lo=f_lo, n_bands=1, n_t=n_t, n_src=3, n_walkers=n_walkers,
                                            amp=(0.1 * amp, amp), n_groups=n_groups, with_data=True)
        nw = d_rows.shape[0]
        buf = np.empty((2 * nw,) + d_rows.shape[1:], np.complex128)
        buf[0::2] = d_rows
        buf[1::2] = d_rows
        cold = tt.tasks["chain_begin"]
        for c in cold:
            buf[2 * tt.chain_walker[c] + 1] = resid[tt.chain_walker[c]]
        tasks = dict(tt.tasks, write_walker=(2 * tt.chain_walker[cold] + 1).astype(np.int32))
        cw2 = (2 * tt.chain_walker).astype(np.int32)
        wpsd = np.repeat(np.arange(nw), 2).astype(np.int32)
        r_ref = buf.copy()
        ref = oracle.temper_sweep(oracle.Config(), oracle.Data(r_ref, wl.psd, wl.k_lo, walker_psd=wpsd), tasks, N, tt.params, cw2,
                                  tt.chain_beta, tt.chain_set_begin, tt.chain_set_n, tt.chain_logu)
        assert ref[1].any()
        d_resid = dev(torch, buf)
        data = gbfit.Data(d_resid, dev(torch, wl.psd), wl.k_lo, walker_psd=dev(torch, wpsd))
        args = [dev(torch, x) for x in (tt.params, cw2, tt.chain_beta, tt.chain_set_begin, tt.chain_set_n, tt.chain_logu)]
        got = ctx.temper_sweep(data, dev(torch, gbfit.pack_temper_tasks(**tasks).view(np.uint8)), N, 3 * N, *args)
        ctx.check()
        perm, acc, dl = (x.cpu().numpy() for x in got)
        assert np.array_equal(acc, ref[1]) and np.array_equal(perm, ref[0])
        assert np.abs(dl - ref[2]).max() <= 1e-6
        r1 = d_resid.cpu().numpy()
        change = np.abs(r_ref - buf).max()
        assert np.abs(r1 - r_ref).max() <= 1e-9 * change + 4e-16 * np.abs(buf).max()
        assert np.array_equal(r1[0::2], buf[0::2])
    # a ladder longer than the odd/even limit: row error, NaN
    t33 = dict(tasks, n_t=np.full_like(tasks["n_t"], 33))
    big = [np.resize(x, (40,) + x.shape[1:]) for x in (cw2, tt.chain_beta, tt.chain_set_begin, tt.chain_set_n, tt.chain_logu)]
    got = ctx.temper_sweep(data, dev(torch, gbfit.pack_temper_tasks(**t33).view(np.uint8)), N, 3 * N, dev(torch, tt.params),
                           *[dev(torch, x) for x in big])
    with pytest.raises(gbfit.GbError):
        ctx.check()
    assert np.isnan(got[2].cpu().numpy()[1:33]).all()
