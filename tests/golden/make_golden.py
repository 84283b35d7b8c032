"""Writes tests/golden/*.txt from the CPU oracle ONLY (never from the CUDA path).

    python tests/golden/make_golden.py

The paper prints no worked example (no flux value, tolerance or iteration count anywhere in
PAPER.md), so these files are REGRESSION fixtures of the oracle on config 1, not paper values:
"parity unpinned" in the sense of DESIGN.md.  The closed-form numbers in closed_forms.txt are
evaluated from formulas derived from eqs. (2)-(7), not from any implementation.
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from oracle import Oracle  # noqa: E402
from workloads import make_problem  # noqa: E402


def main():
    p = make_problem(1)
    for scheme in ("oci", "si"):
        o = Oracle.from_problem(p)
        iters = []
        for k in range(p.n_steps):
            o.set_source(p.source(k))
            st, it, _ = (o.oci_step if scheme == "oci" else o.si_step)(p.tol, p.max_iters)
            iters.append(it)
        hdr = (f"config 1 (BASELINE.json configs[0]) after {p.n_steps} steps, scheme={scheme}, "
               f"tol={p.tol}; iterations per step: {iters}\n"
               "scalar flux phi[j][s], s = (k,L),(k,R),(k+1/2,L),(k+1/2,R); written by "
               "tests/golden/make_golden.py from oracle/ only")
        np.savetxt(os.path.join(HERE, f"cfg1_phi_{scheme}.txt"), o.scalar_flux(), fmt="%.17e", header=hdr)
    z = (2.0 - 1.2) * 1.5 * 0.07
    tau = 1.3 * 0.8 / (1.0 / np.sqrt(3.0))
    with open(os.path.join(HERE, "closed_forms.txt"), "w") as f:
        f.write("# closed forms derived from PAPER.md eqs. (2),(3) [0-D MB decay] and (4),(5) [steady SCB]\n")
        f.write("# name value\n")
        f.write(f"mb_edge_decay_z0.084 {1.0 / (1.0 + z + z * z / 2.0):.17e}\n")
        f.write(f"mb_avg_over_prev_z0.084 {(1.0 + z / 2.0) / (1.0 + z + z * z / 2.0):.17e}\n")
        f.write(f"scb_cell_attenuation_S2_dx0.8_sig1.3 {1.0 / (1.0 + tau + tau * tau / 2.0):.17e}\n")


if __name__ == "__main__":
    main()
