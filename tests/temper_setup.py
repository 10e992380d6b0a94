"""Shared setup of the Algorithm-2 tests: residuals r_t = noise + sum(truth) - sum(set of chain t) on each chain's walker."""
import numpy as np


def temper_case(oracle, N=128, f_lo=6e-4, n_bands=3, n_t=4, n_src=3, n_walkers=5, amp=(2e-23, 2e-22), jitter=1.0, stream=0,
                n_groups=1, with_data=False):
    """with_data: also return the DATA rows d_w = noise + sum of the true sources of the ladders walker w takes part in
    (the rows the odd/even buffer mode stages from: they hold none of the chains' own sets)."""
    from gb_inputs import make_workload, make_temper_tasks
    wl = make_workload(3, B=1, n_walkers=n_walkers)
    tt = make_temper_tasks(wl, N, f_lo, n_bands, n_t, n_src, stream=stream, amp_lo=amp[0], amp_hi=amp[1], jitter=jitter,
                           n_groups=n_groups)
    resid = wl.resid()
    cfg = oracle.Config()
    data = oracle.Data(resid, wl.psd, wl.k_lo)
    for it in range(len(tt.tasks["n_t"])):
        for t in range(n_t):
            c = tt.tasks["chain_begin"][it] + t
            w = np.full(1, tt.chain_walker[c], np.int32)
            for src in tt.truth[it // n_groups]:          # the data hold the true sources: r = d - H
                oracle.residual_update(cfg, data, None, src[None], w, move_all=oracle.REMOVE, N=N)
    d_rows = resid.copy() if with_data else None
    for it in range(len(tt.tasks["n_t"])):
        for t in range(n_t):
            c = tt.tasks["chain_begin"][it] + t
            w = np.full(1, tt.chain_walker[c], np.int32)
            for src in tt.params[tt.chain_set_begin[c]:tt.chain_set_begin[c] + tt.chain_set_n[c]]:
                oracle.residual_update(cfg, data, src[None], None, w, move_all=oracle.ADD, N=N)
    return (wl, tt, resid, d_rows) if with_data else (wl, tt, resid)
