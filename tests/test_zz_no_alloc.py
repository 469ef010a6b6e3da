"""afqmc_comb_map_noalloc: the allocation-free variant of afqmc_comb_map (scratch in a file-scope device array of
AFQMC_NOALLOC_MAX_WALKERS doubles) against the existing path with caller-provided scratch, on two calls in a row.  The
parent map is an integer decision taken in FP64 from the same weights, so -- as in the other comb tests -- the comparison
is bit-exact, also against the oracle's map.  Collected last on purpose (file name): the suite runs with pytest -x."""
import numpy as np
import pytest

from oracle import afqmc_oracle as orc
from workloads import make_workload

from . import gpu_harness as H

pytestmark = pytest.mark.gpu

MAXW = 65536        # AFQMC_NOALLOC_MAX_WALKERS in include/afqmc.h


def _both(ctx, w, u):
    import torch
    dev = ctx.device
    n = w.shape[0]
    wd = torch.tensor(w, dtype=torch.float64, device=dev)
    cum = torch.empty(n, dtype=torch.float64, device=dev)
    par_a = torch.full((n,), -1, dtype=torch.int32, device=dev)
    par_b = torch.full((n,), -2, dtype=torch.int32, device=dev)
    wn_a = torch.zeros(2, dtype=torch.float64, device=dev)
    wn_b = torch.ones(2, dtype=torch.float64, device=dev)
    ctx.afqmc_comb_map(wd, u, cum, par_a, wn_a)              # existing path: caller-provided scratch
    ctx.afqmc_comb_map_noalloc(wd, u, par_b, wn_b)           # new path: the library's static scratch
    torch.cuda.synchronize()
    return par_a.cpu().numpy(), wn_a.cpu().numpy(), par_b.cpu().numpy(), wn_b.cpu().numpy()


def test_comb_map_noalloc_matches_existing_path_twice_in_a_row():
    import torch
    import paper_1804_03310_b200 as afq
    wl = make_workload(1, "tame")
    ctx = H.make_ctx(wl, 8)
    rng = np.random.default_rng(123)
    # call 1: a large population (leaves the static array full of running sums); call 2: a smaller one with dead walkers,
    # which must not see anything of call 1; call 3: the maximum size
    cases = [(rng.random(3001) ** 3, 0.37), (np.where(rng.random(777) < 0.3, 0.0, rng.random(777)), 0.999999),
             (np.exp(0.5 * rng.standard_normal(MAXW)), 0.0)]
    mem0 = torch.cuda.memory_allocated(ctx.device)
    for w, u in cases:
        pa, wa, pb, wb = _both(ctx, w, u)
        assert np.array_equal(pa, pb)
        assert np.array_equal(wa, wb)
        assert np.array_equal(pb, orc.o_comb(w, u))
        assert wb[0] == np.cumsum(w)[-1] / w.shape[0]
    # a dead population: identity map, weights kept (w_new[0] = -1), as the existing path
    pa, wa, pb, wb = _both(ctx, np.zeros(33), 0.5)
    assert np.array_equal(pb, np.arange(33)) and np.array_equal(pa, pb) and wb[0] == -1.0 == wa[0]
    # sizes beyond the static scratch are rejected before any launch, with a clear error
    l0 = ctx.launch_count
    big = torch.ones(MAXW + 1, dtype=torch.float64, device=ctx.device)
    par = torch.zeros(MAXW + 1, dtype=torch.int32, device=ctx.device)
    wn = torch.zeros(2, dtype=torch.float64, device=ctx.device)
    with pytest.raises(afq.AfqmcError) as ei:
        ctx.afqmc_comb_map_noalloc(big, 0.5, par, wn)
    assert ei.value.status == afq.AFQMC_EUNSUPPORTED and "AFQMC_NOALLOC_MAX_WALKERS" in str(ei.value)
    with pytest.raises(afq.AfqmcError):
        ctx.afqmc_comb_map_noalloc(big[:10], 1.0, par, wn)
    assert ctx.launch_count == l0
    del big, par, wn
    assert torch.cuda.memory_allocated(ctx.device) <= mem0 + (1 << 20)      # nothing was allocated on our behalf
