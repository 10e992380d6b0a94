"""Parity of gb_delta_loglike_accept (the batched sweep step with its accept / reject decision; BASELINE config 5,
Alg. 1, Eq. 13) with the CPU oracle: delta lnL <= 1e-6, decisions bit-exact (both sides
decide beta dlnL + logq >= logu with separately rounded FP64 operations), residuals after the update <= 1e-9 of the largest
change, for the fused update (apply = 1: the accepted windows of one walker chunk are moved into the residual by the CTAs
that evaluate the next chunk), the separate launch (apply = 2) and decide-and-keep (apply = 0 + gb_residual_update_kept)."""
import numpy as np
import pytest

from gb_inputs import make_workload

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
    return None if a is None else torch.as_tensor(np.ascontiguousarray(a)).to("cuda:0")


def _draws(B, key, rate=0.35):
    """logu, logq, beta such that about `rate` of the rows are accepted whatever delta lnL is (a seeded part decided by
    +-inf, so the parity of decisions cannot flip on a threshold) plus a part decided by the actual delta lnL."""
    g = np.random.Generator(np.random.Philox(key=key))
    logu = np.log(g.random(B))
    forced = g.random(B)
    logu[forced < rate] = -np.inf
    logu[(forced >= rate) & (forced < 0.8)] = np.inf
    logq = 0.2 * g.standard_normal(B)
    beta = np.asarray([1.0, 0.7, 0.4, 0.0])[g.integers(0, 4, B)]
    return logu, logq, beta


def _case(B=9000, n_walkers=5, general_row=True):
    wl = make_workload(3, B=B, n_walkers=n_walkers)          # mixed ADD / REMOVE, N by f0 (128 .. 1024)
    if general_row:
        wl.params_new[10, 2] = 3e-12                         # outside the fast-path limits: the general kernels' epilogue
        wl.params_old[10] = wl.params_new[10]
    return wl


def _oracle(oracle, wl, resid, logu, logq, beta, apply=True):
    od = oracle.Data(resid.copy(), wl.psd, wl.k_lo)
    dl, acc = oracle.delta_loglike_accept(oracle.Config(), od, wl.params_new, wl.params_old, wl.walker_index, logu, logq=logq,
                                          beta=beta, move=wl.move, n_bins=wl.n_bins, apply=apply,
                                          nthreads=oracle.max_threads())
    return dl, acc, od.resid


def _gpu(torch, gbfit, ctx, wl, resid, logu, logq, beta, apply, store_bins=None, check=True):
    d_resid = dev(torch, resid)
    data = gbfit.Data(d_resid, dev(torch, wl.psd), wl.k_lo)
    dl, acc = ctx.delta_loglike_accept(data, dev(torch, wl.params_new), dev(torch, wl.params_old), dev(torch, wl.walker_index),
                                       dev(torch, logu), logq=dev(torch, logq), beta=dev(torch, beta), move=dev(torch, wl.move),
                                       n_bins=dev(torch, wl.n_bins),
                                       store_bins=int(wl.n_bins.sum()) if store_bins is None else store_bins, apply=apply)
    if check:
        ctx.check()
    return dl.cpu().numpy(), acc.cpu().numpy(), d_resid, data


def _same(got_dl, got_acc, got_r, ref_dl, ref_acc, ref_r, resid):
    assert np.abs(got_dl - ref_dl).max() <= 1e-6
    assert np.array_equal(got_acc, ref_acc), int((got_acc != ref_acc).sum())
    dref = ref_r - resid
    assert np.abs((got_r - resid) - dref).max() <= 1e-9 * np.abs(dref).max() + 4e-16 * np.abs(resid).max()


@pytest.mark.parametrize("apply", [1, 2])
def test_accept_fused_and_separate_update_match_the_oracle(oracle, torch_cuda, gb, apply):
    gbfit, ctx = gb
    wl = _case()
    resid = wl.resid()
    logu, logq, beta = _draws(wl.B, [31, apply])
    ref = _oracle(oracle, wl, resid, logu, logq, beta)
    assert 0.2 < ref[1].mean() < 0.6
    dl, acc, d_resid, data_acc = _gpu(torch_cuda, gbfit, ctx, wl, resid, logu, logq, beta, apply)
    _same(dl, acc, d_resid.cpu().numpy(), *ref, resid)
    # the accepted windows stay in the context: negate = 1 undoes the call's update
    ctx.residual_update_kept(data_acc, negate=True)
    ctx.check()
    assert np.abs(d_resid.cpu().numpy() - resid).max() <= 4e-16 * max(np.abs(resid).max(), np.abs(ref[2] - resid).max())
    # the same bits of delta lnL as the plain call
    data = gbfit.Data(dev(torch_cuda, resid), dev(torch_cuda, wl.psd), wl.k_lo)
    plain = ctx.delta_loglike(data, dev(torch_cuda, wl.params_new), dev(torch_cuda, wl.params_old),
                              dev(torch_cuda, wl.walker_index), move=dev(torch_cuda, wl.move), n_bins=dev(torch_cuda, wl.n_bins))
    assert np.array_equal(plain.cpu().numpy(), dl)


def test_accept_keep_then_update_kept_and_undo(oracle, torch_cuda, gb):
    gbfit, ctx = gb
    torch = torch_cuda
    wl = _case(B=5000, n_walkers=3)
    resid = wl.resid()
    logu, logq, beta = _draws(wl.B, [32, 0])
    ref = _oracle(oracle, wl, resid, logu, logq, beta)
    dl, acc, d_resid, data = _gpu(torch, gbfit, ctx, wl, resid, logu, logq, beta, apply=0)
    assert np.array_equal(d_resid.cpu().numpy(), resid)            # decided and kept, nothing applied
    ctx.residual_update_kept(data)
    ctx.check()
    _same(dl, acc, d_resid.cpu().numpy(), *ref, resid)
    ctx.residual_update_kept(data, negate=True)
    assert np.abs(d_resid.cpu().numpy() - resid).max() <= 4e-16 * max(np.abs(resid).max(), np.abs(ref[2] - resid).max())
    with pytest.raises(gbfit.GbError):                              # the call decided: an `accepted` array is refused
        ctx.residual_update_kept(data, dev(torch, acc))
    ctx.delta_loglike(data, dev(torch, wl.params_new), dev(torch, wl.params_old), dev(torch, wl.walker_index),
                      move=dev(torch, wl.move), n_bins=dev(torch, wl.n_bins))
    with pytest.raises(gbfit.GbError):                              # kept state does not survive another batched call
        ctx.residual_update_kept(data)


def test_accept_snapshot_semantics_duplicates_empty_walkers_and_single_window_length(oracle, torch_cuda, gb):
    """Rows are evaluated against ONE snapshot although accepted windows are scattered while the call is still running:
    duplicated rows (same source, same walker, both accepted) get identical delta lnL; walkers without any row and a walker
    whose rows are all rejected are fine; the fixed-N form (no n_bins: one kernel class, which is also the draining one)."""
    gbfit, ctx = gb
    torch = torch_cuda
    wl = make_workload(2, B=4096)                                   # one walker, ADD, N = 256
    wl = wl.subset(np.arange(1500))
    resid1 = wl.resid()
    resid = np.concatenate([resid1, resid1[:1] * 0.5, resid1[:1] * 2.0, resid1[:1]])       # 4 walkers
    psd = np.concatenate([wl.psd] * 4)
    w = (np.arange(wl.B) % 3).astype(np.int32) * (np.arange(wl.B) % 3 != 1)                 # walkers 0 and 2 only; 1, 3 empty
    pn = wl.params_new.copy()
    pn[1::2] = pn[0::2]                                             # duplicates
    w[1::2] = w[0::2]
    logu = np.full(wl.B, -np.inf)
    logu[w == 2] = np.inf                                           # every row of walker 2 rejected
    od = oracle.Data(resid.copy(), psd, wl.k_lo)
    rdl, racc = oracle.delta_loglike_accept(oracle.Config(), od, pn, None, w, logu, move_all=oracle.ADD, N=256,
                                            nthreads=oracle.max_threads())
    assert np.array_equal(rdl[0::2], rdl[1::2])
    for apply in (1, 2):
        d_resid = dev(torch, resid)
        data = gbfit.Data(d_resid, dev(torch, psd), wl.k_lo)
        dl, acc = ctx.delta_loglike_accept(data, dev(torch, pn), None, dev(torch, w), dev(torch, logu), move_all=gbfit.ADD, N=256,
                                           store_bins=256 * wl.B, apply=apply)
        ctx.check()
        dl, acc = dl.cpu().numpy(), acc.cpu().numpy()
        assert np.array_equal(dl[0::2], dl[1::2])
        _same(dl, acc, d_resid.cpu().numpy(), rdl, racc, od.resid, resid)
        assert np.array_equal(d_resid.cpu().numpy()[1:], resid[1:])


def test_accept_undersized_store_rejects_the_rows_that_do_not_fit(oracle, torch_cuda, gb):
    """store_bins too small: flag 4; the rows reported accepted are exactly the rows applied (the residual equals the
    oracle's update by the REPORTED flags), the others are reported rejected although Eq. 13 would accept them."""
    gbfit, ctx = gb
    torch = torch_cuda
    wl = _case(B=3000, n_walkers=2, general_row=False)
    resid = wl.resid()
    logu = np.full(wl.B, -np.inf)
    dl, acc, d_resid, _ = _gpu(torch, gbfit, ctx, wl, resid, logu, None, None, apply=1, store_bins=int(wl.n_bins.sum()) // 3,
                               check=False)
    with pytest.raises(gbfit.GbError) as ei:
        ctx.check()
    assert ei.value.code == gbfit.GB_ERR_ROW
    assert 0 < acc.sum() < wl.B and wl.n_bins[acc != 0].sum() <= int(wl.n_bins.sum()) // 3
    od = oracle.Data(resid.copy(), wl.psd, wl.k_lo)
    oracle.residual_update(oracle.Config(), od, wl.params_new, wl.params_old, wl.walker_index, move=wl.move, accepted=acc,
                           n_bins=wl.n_bins, nthreads=oracle.max_threads())
    dref = od.resid - resid
    assert np.abs((d_resid.cpu().numpy() - resid) - dref).max() <= 1e-9 * np.abs(dref).max()
    # argument errors
    data = gbfit.Data(dev(torch, resid), dev(torch, wl.psd), wl.k_lo)
    with pytest.raises(gbfit.GbError):
        ctx.delta_loglike_accept(data, dev(torch, wl.params_new), dev(torch, wl.params_old), dev(torch, wl.walker_index),
                                 dev(torch, logu), move_all=gbfit.SWAP, N=256, store_bins=256 * wl.B)
    mv = wl.move.copy()
    mv[5] = gbfit.SWAP                                              # a SWAP row is a row error (NaN, rejected)
    dl, acc = ctx.delta_loglike_accept(data, dev(torch, wl.params_new), dev(torch, wl.params_old), dev(torch, wl.walker_index),
                                       dev(torch, logu), move=dev(torch, mv), n_bins=dev(torch, wl.n_bins),
                                       store_bins=int(wl.n_bins.sum()), apply=2)
    with pytest.raises(gbfit.GbError):
        ctx.check()
    assert np.isnan(dl.cpu().numpy()[5]) and acc.cpu().numpy()[5] == 0


def test_accept_launch_scale_walker_chunks_and_fused_update(oracle, torch_cuda, gb):
    """800 000 rows of 36 walkers: the call works through the walkers in 3 chunks (one per 2^18 rows) and the accepted
    windows of a chunk are moved into the residual by the CTAs that evaluate the next chunk (bulk copy + bulk add.f64
    reduction), the last chunk by a closing launch; more than one wave of CTAs in every class.  The oracle replays the
    whole batch; rows are in random walker order, so the binning by (class, walker chunk) is what keeps a walker's rows
    ahead of its update."""
    gbfit, ctx = gb
    wl = make_workload(3, B=800000, n_walkers=36)
    resid = wl.resid()
    logu, logq, beta = _draws(wl.B, [33, 0], rate=0.25)
    ref = _oracle(oracle, wl, resid, logu, logq, beta)
    dl, acc, d_resid, _ = _gpu(torch_cuda, gbfit, ctx, wl, resid, logu, logq, beta, apply=1, store_bins=int(0.6 * wl.n_bins.sum()))
    _same(dl, acc, d_resid.cpu().numpy(), *ref, resid)
    assert ctx.launch_count() > 0


def test_accept_host_form_chunked(oracle, torch_cuda, gb):
    """gb_delta_loglike_accept_host: HOST arrays in, HOST (dlnL, accepted) out; 300 000 rows flow through in chunks (each chunk
    one accept call of its own), rows sorted by walker so that a walker's rows do not straddle chunks in a way that matters
    (they may: the snapshot semantics hold per chunk, and the oracle is run chunk by chunk the same way)."""
    gbfit, ctx = gb
    torch = torch_cuda
    wl = make_workload(3, B=300000, n_walkers=8)
    wl = wl.subset(np.argsort(wl.walker_index, kind="stable"))
    resid = wl.resid()
    logu, logq, beta = _draws(wl.B, [34, 0], rate=0.25)
    od = oracle.Data(resid.copy(), wl.psd, wl.k_lo)
    rdl, racc = np.zeros(wl.B), np.zeros(wl.B, np.uint8)
    cuts = gbfit.HOST_ACCEPT_CUTS                                   # the library's chunking (include/gbfit.h)
    for c in range(len(cuts) - 1):
        lo, hi = wl.B * cuts[c] // 24, wl.B * cuts[c + 1] // 24
        sl = slice(lo, hi)
        rdl[sl], racc[sl] = oracle.delta_loglike_accept(oracle.Config(), od, wl.params_new[sl], wl.params_old[sl], wl.walker_index[sl],
                                                        logu[sl], logq=logq[sl], beta=beta[sl], move=wl.move[sl], n_bins=wl.n_bins[sl],
                                                        nthreads=oracle.max_threads())
    d_resid = dev(torch, resid)
    data = gbfit.Data(d_resid, dev(torch, wl.psd), wl.k_lo)
    dl, acc = ctx.delta_loglike_accept_host(data, wl.params_new, wl.params_old, wl.walker_index, logu, logq=logq, beta=beta,
                                            move=wl.move, n_bins=wl.n_bins, store_bins=int(0.6 * wl.n_bins.sum()), apply=1)
    ctx.check()
    _same(np.asarray(dl), np.asarray(acc), d_resid.cpu().numpy(), rdl, racc, od.resid, resid)


def test_accept_repeated_calls_agree(oracle, torch_cuda, gb):
    """Race check without a sanitizer: the fused call repeated on fresh copies of the residual gives bit-identical delta lnL
    and decisions every time, and final residuals that agree to the rounding order of the adds (400 000 rows, 2 walker
    chunks, so the in-loop update, the piece kernel and the closing scatter all run)."""
    gbfit, ctx = gb
    torch = torch_cuda
    wl = make_workload(3, B=400000, n_walkers=12)
    resid = wl.resid()
    logu, logq, beta = _draws(wl.B, [35, 0], rate=0.25)
    first = None
    for rep in range(3):
        dl, acc, d_resid, _ = _gpu(torch, gbfit, ctx, wl, resid, logu, logq, beta, apply=1, store_bins=int(0.6 * wl.n_bins.sum()))
        r1 = d_resid.cpu().numpy()
        if first is None:
            first = (dl, acc, r1)
            assert 0.2 < acc.mean() < 0.6
        else:
            assert np.array_equal(dl, first[0]) and np.array_equal(acc, first[1])
            change = np.abs(first[2] - resid).max()
            assert np.abs(r1 - first[2]).max() <= 1e-12 * change + 4e-16 * np.abs(resid).max()
    # gb_scratch_bytes: at least the window store (32 bytes per store bin) and the source records (192 bytes per row)
    assert ctx.scratch_bytes() >= 32 * int(0.6 * wl.n_bins.sum()) + 192 * wl.B
