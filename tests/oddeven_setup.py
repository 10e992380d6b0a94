"""Shared setup of the odd/even cold-chain buffer tests (Fig. 4).

Rows of the residual array: 2 w = EVEN buffer of walker w (data minus the cold-chain sources of even sub-bands),
2 w + 1 = ODD buffer (data minus the cold-chain sources of odd sub-bands).  Tasks run the ODD sub-bands: they stage
from the even buffer, subtract their own current sources online, and the cold chain writes back into the odd buffer.
"""
import numpy as np


def oddeven_case(oracle, N=128, f_lo=6e-4, n_bands=3, n_src=3, n_prop=10, n_walkers=2, amp=(2e-23, 2e-22)):
    from gb_inputs import make_workload, make_band_tasks
    wl = make_workload(3, B=1, n_walkers=n_walkers)
    cold = make_band_tasks(wl, N, f_lo, n_bands, n_src, n_prop, stream=10, amp_lo=amp[0], amp_hi=amp[1])
    hot = make_band_tasks(wl, N, f_lo, n_bands, n_src, n_prop, stream=11, amp_lo=amp[0], amp_hi=amp[1], betas=(0.5, 0.7))
    cfg = oracle.Config()
    d = wl.resid()                                                  # the data of each walker
    # cold-chain sources of the even sub-bands 0, 2, .., 2 n_bands (seeded here: plain inputs)
    g = np.random.Generator(np.random.Philox(key=[2405, N]))
    kb0 = int(cold.tasks["k_first"][0])                             # first bin of sub-band 0
    n_even = n_bands + 1
    u = g.random((n_walkers, n_even, 2, 8))
    ev = np.empty_like(u)
    ev[..., 0] = amp[0] * (amp[1] / amp[0]) ** u[..., 0]
    ev[..., 1] = (kb0 + (2 * np.arange(n_even)[None, :, None] + u[..., 1]) * N) / wl.Tobs
    ev[..., 2] = 0.0
    ev[..., 3] = 2 * np.pi * u[..., 3]
    ev[..., 4] = 1.8 * u[..., 4] - 0.9
    ev[..., 5] = np.pi * u[..., 5]
    ev[..., 6] = 2 * np.pi * u[..., 6]
    ev[..., 7] = 1.8 * u[..., 7] - 0.9
    buf = np.empty((2 * n_walkers, 2, wl.n_f), np.complex128)
    buf[0::2] = d
    buf[1::2] = d
    data = oracle.Data(buf, wl.psd, wl.k_lo, walker_psd=np.repeat(np.arange(n_walkers), 2).astype(np.int32))
    for w in range(n_walkers):
        for src in ev[w].reshape(-1, 8):                            # even buffer: minus the even bands' cold sources
            oracle.residual_update(cfg, data, src[None], None, np.full(1, 2 * w, np.int32), move_all=oracle.ADD, N=N)
    t = cold.tasks
    for i in range(len(t["walker"])):                               # odd buffer: minus the odd bands' cold sources
        for src in cold.params[t["src_begin"][i]:t["src_begin"][i] + t["n_src"][i]]:
            oracle.residual_update(cfg, data, src[None], None, np.full(1, 2 * t["walker"][i] + 1, np.int32),
                                   move_all=oracle.ADD, N=N)

    def remap(bt, cold_chain):
        tt = {k: v.copy() for k, v in bt.tasks.items()}
        w = tt["walker"].copy()
        tt["walker"] = (2 * w).astype(np.int32)                     # stage from the EVEN buffer
        tt["subtract_current"] = np.ones_like(w)
        tt["write_walker"] = (2 * w + 1).astype(np.int32)           # the cold chain updates the ODD buffer
        tt["write_back"] = np.full_like(w, 1 if cold_chain else 0)
        return tt

    return wl, d, buf, data.walker_psd, cold, remap(cold, True), hot, remap(hot, False), ev
