"""gb_band_sweep_static, the entry point that allocates nothing (include/gbfit.h): its kernel's scratch is the library's
file-scope device array instead of context-owned cudaMalloc memory.  Two calls in a row (different window lengths, so the
second one finds the first one's contents in the array) are compared with the existing path, gb_band_sweep, on the same
seeded band tasks: decisions and final parameters bit-exact, delta lnL <= 1e-6 absolute, final residuals <= 1e-9 of the
largest change (the tolerances of test_gpu_band_sweep.py).  Also: the free device memory does not move across the calls,
and a call beyond GB_STATIC_MAX_TASK_BINS is refused.

This file is named so that pytest collects it last: the suite runs with `pytest -x`.
"""
import numpy as np
import pytest

from gb_inputs import make_band_tasks, make_workload

pytestmark = pytest.mark.gpu

TOL_DLNL = 1e-6
CASES = ((256, 2e-3, 6, 2e-22), (1024, 1.2e-2, 3, 1e-23))   # (N, f_lo, bands per walker, largest amplitude)


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


class Case:
    """Device copies of one seeded band-sweep problem, every output preallocated (the static call must not need any)."""

    def __init__(self, torch, gbfit, N, f_lo, n_bands, amp, stream):
        self.N = N
        self.wl = make_workload(3, B=1, n_walkers=3)
        self.bt = make_band_tasks(self.wl, N, f_lo, n_bands, n_src=5, n_prop=14, amp_lo=0.1 * amp, amp_hi=amp, stream=stream)
        self.resid0 = self.wl.resid()
        self.n_tasks = int(self.bt.tasks["walker"].shape[0])
        self.max_stage = int(self.bt.tasks["n_stage"].max())
        self.tasks = dev(torch, gbfit.pack_band_tasks(**self.bt.tasks).view(np.uint8))
        self.psd = dev(torch, self.wl.psd)
        self.prop = [dev(torch, a) for a in (self.bt.prop_k, self.bt.prop_params, self.bt.prop_logq, self.bt.prop_logu)]
        P = int(self.bt.prop_k.shape[0])
        self.resid = dev(torch, self.resid0)
        self.params = dev(torch, self.bt.params)
        self.acc = torch.zeros((P,), dtype=torch.uint8, device="cuda:0")
        self.dl = torch.zeros((P,), dtype=torch.float64, device="cuda:0")
        self.data = gbfit.Data(self.resid, self.psd, self.wl.k_lo)

    def reset(self, torch):
        self.resid.copy_(torch.as_tensor(self.resid0))
        self.params.copy_(torch.as_tensor(self.bt.params))
        self.acc.zero_()
        self.dl.fill_(float("nan"))

    def run(self, ctx, static):
        fn = ctx.band_sweep_static if static else ctx.band_sweep
        fn(self.data, self.tasks, self.N, self.max_stage, self.params, *self.prop, accepted_out=self.acc, dlnL_out=self.dl)

    def result(self):
        return self.acc.cpu().numpy(), self.dl.cpu().numpy(), self.params.cpu().numpy(), self.resid.cpu().numpy()


def compare(got, ref, resid0):
    acc, dl, params, r1 = got
    racc, rdl, rparams, rr1 = ref
    assert 0 < racc.sum() < racc.size                      # a mix of accepted and rejected proposals
    assert np.array_equal(acc, racc), int((acc != racc).sum())
    assert np.isfinite(rdl).all() and np.abs(dl - rdl).max() <= TOL_DLNL
    assert np.array_equal(params, rparams)
    change = np.abs(rr1 - resid0).max()
    assert change > 0
    assert np.abs(r1 - rr1).max() <= 1e-9 * change + 4e-16 * np.abs(resid0).max()


def test_band_sweep_static_matches_band_sweep_two_calls_in_a_row(torch_cuda, gb):
    torch = torch_cuda
    gbfit, ctx = gb
    cases = [Case(torch, gbfit, *c, stream=7 + i) for i, c in enumerate(CASES)]
    for c in cases:
        assert c.n_tasks * c.N <= gbfit.STATIC_MAX_TASK_BINS

    # the existing path (context-owned scratch from cudaMalloc) gives the expected values
    ref = []
    for c in cases:
        c.reset(torch)
        c.run(ctx, static=False)
        ctx.check()
        ref.append(c.result())

    # once untimed and unchecked, so that what the driver sets up at a kernel's first launch is in place
    for c in cases:
        c.reset(torch)
        c.run(ctx, static=True)
    for c in cases:
        c.reset(torch)
    torch.cuda.synchronize()

    # two calls in a row on one stream; the second finds the array as the first left it
    free0 = torch.cuda.mem_get_info(0)[0]
    for c in cases:
        c.run(ctx, static=True)
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info(0)[0]
    ctx.check()
    assert free1 == free0, (free0, free1)                   # no device memory was taken or given back
    for c, r in zip(cases, ref):
        compare(c.result(), r, c.resid0)

    # and once more in the other order
    for c in cases:
        c.reset(torch)
    for c in reversed(cases):
        c.run(ctx, static=True)
    ctx.check()
    for c, r in zip(cases, ref):
        compare(c.result(), r, c.resid0)


def test_band_sweep_static_refuses_sizes_beyond_the_static_array(torch_cuda, gb):
    torch = torch_cuda
    gbfit, ctx = gb
    N = 1024
    c = Case(torch, gbfit, N, 1.2e-2, 11, 1e-23, stream=9)   # 33 tasks of N = 1024: one more than the array holds
    assert c.n_tasks * N > gbfit.STATIC_MAX_TASK_BINS
    c.reset(torch)
    before = c.result()
    with pytest.raises(gbfit.GbError, match="GB_STATIC_MAX_TASK_BINS"):
        c.run(ctx, static=True)
    torch.cuda.synchronize()
    after = c.result()
    assert np.array_equal(before[0], after[0]) and np.array_equal(before[2], after[2]) and np.array_equal(before[3], after[3])
    ctx.check()
    # the same problem is fine on the allocating path
    c.run(ctx, static=False)
    ctx.check()
    assert np.isfinite(c.result()[1]).all()
