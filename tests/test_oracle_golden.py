"""Regression of the oracle against stored fixtures (see tests/golden/make_golden.py)."""
import os

import numpy as np

from oracle import Oracle
from workloads import make_problem

G = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def test_cfg1_regression():
    p = make_problem(1)
    for scheme, iters in (("oci", 7), ("si", 8)):
        o = Oracle.from_problem(p)
        for k in range(p.n_steps):
            o.set_source(p.source(k))
            st, it, _ = (o.oci_step if scheme == "oci" else o.si_step)(p.tol, p.max_iters)
            assert st == 0 and it == iters
        ref = np.loadtxt(os.path.join(G, f"cfg1_phi_{scheme}.txt"))
        assert np.max(np.abs(o.scalar_flux() - ref)) <= 1e-15


def test_closed_form_fixture_values():
    vals = dict(line.split() for line in open(os.path.join(G, "closed_forms.txt")) if not line.startswith("#"))
    assert abs(float(vals["mb_edge_decay_z0.084"]) - 0.9195165549760558) < 1e-15
    assert abs(float(vals["mb_avg_over_prev_z0.084"]) - 0.9581362502850501) < 1e-15
    assert abs(float(vals["scb_cell_attenuation_S2_dx0.8_sig1.3"]) - 0.2260534341013726) < 1e-15
