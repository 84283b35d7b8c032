"""Fig. 1-style spectral-radius map from the CPU oracle: rho(OCI), rho(SI) and their ratio over the
cell optical thickness Sigma*dx and the scattering ratio c, for the steady problem (dt -> infinity), S4 Gauss-Legendre,
infinite medium via reflecting boundaries - the setting the paper states for its figure (whose values are an image that
is not available, so this table is the oracle's own result, not a reproduction of printed numbers).

    python -m oracle.rho_map [--cells 24] [--out oracle/rho_map_S4.txt]

Method: power iteration on the homogeneous problem (Q = 0, psi_{k-1/2} = 0, so the iterate IS the error): rho is the
geometric-mean contraction of max|phi^(l+1) - phi^(l)| over the second half of the iterations.  TEST INFRASTRUCTURE:
calls only oracle/."""
import argparse
import sys

import numpy as np

from . import Oracle

THICK = (0.05, 0.1, 0.25, 0.5, 1.0, 2.0, 5.0, 10.0)
CS = (0.5, 0.8, 0.9, 0.99)


def rho(scheme, thick, c, cells, N=4, seed=3):
    o = Oracle(np.full(cells, thick), np.ones(cells), np.full(cells, c), 1.0, 1e12, N, (2, 0.0), (2, 0.0))
    o.setup()
    o.set_flux(np.zeros((cells, N, 2)))
    o.set_source(None)
    o.set_iterate(np.random.default_rng(seed).uniform(0.5, 1.5, (cells, 4 * N)))
    f = o.oci_iteration if scheme == "oci" else o.si_iteration
    # enough iterations for the slowest mode to dominate, few enough not to underflow: stop at 1e-200
    ds = []
    for _ in range(4000 if scheme == "oci" else 400):
        d, _ = f()
        if d < 1e-200:
            break
        ds.append(d)
    ds = np.array(ds)
    half = len(ds) // 2
    return (ds[-1] / ds[half]) ** (1.0 / (len(ds) - 1 - half))


def table(cells):
    lines = ["# rho(OCI), rho(SI), rho(OCI)/rho(SI): steady (dt = 1e12), S4, reflecting/reflecting, %d cells, Sigma = 1" % cells,
             "# rows: Sigma*dx; columns: c = " + ", ".join(f"{c:g}" for c in CS),
             "# written by `python -m oracle.rho_map` (oracle only); cf. PAPER.md:31-37, Fig. 1"]
    grid = {}
    for th in THICK:
        cells_txt = []
        for c in CS:
            a, b = rho("oci", th, c, cells), rho("si", th, c, cells)
            grid[(th, c)] = (a, b)
            cells_txt.append(f"{a:.4f} {b:.4f} {a / b:6.3f}")
        lines.append(f"{th:5.2f} | " + " | ".join(cells_txt))
    return "\n".join(lines) + "\n", grid


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--cells", type=int, default=24)
    ap.add_argument("--out", default=None)
    a = ap.parse_args()
    txt, _ = table(a.cells)
    sys.stdout.write(txt)
    if a.out:
        with open(a.out, "w") as f:
            f.write(txt)


if __name__ == "__main__":
    main()
