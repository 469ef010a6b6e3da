"""Host-side pieces of bench.py that run without a GPU: the `cpu_baseline` / `--impl reference` leg (the oracle timed on a
bounded sample).  Regression: on a multi-determinant workload the workload's own initial walkers are the reference
determinant, whose overlap with every excited determinant is exactly zero, and the oracle's SMW path raised
LinAlgError on the exactly singular matrix -- `python bench.py --cfg 4` died in its CPU-baseline leg."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


@pytest.mark.parametrize("cfg", [2, 4])
def test_time_oracle_runs_on_single_and_multi_determinant_workloads(cfg):
    import bench
    from workloads import make_workload
    wl = make_workload(cfg, "mf")
    out = bench.time_oracle(wl, target_s=0.2, one_thread_s=0.0)
    assert out["kind"] == "oracle" and out["unit"] == bench.UNIT
    assert np.isfinite(out["value"]) and out["value"] > 0
    assert ("reference determinant" in out["sample"]) == (wl.n_det > 1)
