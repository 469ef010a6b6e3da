"""Writes tests/golden/cfg1_raw_10steps.txt from the FP64 oracle ONLY (oracle/ + workloads/; nothing from the CUDA
path).  The paper prints no step-level worked example, so this fixture is not a paper value: it
freezes the oracle's own trajectory on BASELINE.json config 1 so that any later change to the oracle's arithmetic is
visible in review (tests/test_oracle_pins.py::test_oracle_trajectory_fixture).
Run:  python tests/golden/write_oracle_fixture.py"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import afqmc_oracle as orc  # noqa: E402
from workloads import make_workload  # noqa: E402


def trajectory():
    wl = make_workload(1, "raw")
    ini = orc.o_init(wl.h, wl.L, wl.dt, wl.psi_a, wl.psi_b)
    st = orc.o_seed_state(ini, wl.walkers(), wl.n_alpha)
    xs = wl.fields()
    rows = []
    for n in range(wl.steps):
        st, rec = orc.o_step(ini, st, xs[n], wl.n_alpha, K=wl.K, E0=wl.E0)
        rows.append((n + 1, orc.o_mixed_energy(st.w, st.eloc), float(np.sum(st.w)), int(np.sum(st.w > 0)),
                     st.S[0].real, st.S[0].imag, st.eloc[0].real, st.eloc[0].imag))
    return rows


if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg1_raw_10steps.txt")
    with open(out, "w") as f:
        f.write("# BASELINE.json config 1 (raw), FP64 oracle, hybrid weights, E0 = 0; written by write_oracle_fixture.py\n")
        f.write("# step  E_mix  sum_w  n_alive  Re S[0]  Im S[0]  Re E_L[0]  Im E_L[0]\n")
        for r in trajectory():
            f.write("%d %.15e %.15e %d %.15e %.15e %.15e %.15e\n" % r)
    print("wrote", out)
