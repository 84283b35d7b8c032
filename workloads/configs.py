"""The five BASELINE.json configs as concrete, seeded, synthetic inputs.

Recipe: SURVEY.md §8(d) "Inputs" table (restated in DESIGN.md §Inputs).  The
paper uses no public dataset; its timed workloads are a Reed-type multi-region
slab and a homogeneous 10-cm slab sweep.  These
five configs are synthetic stand-ins shaped like the latter.

Layouts (all float64, C-contiguous):
  dx, sigma_t, sigma_s : [J]
  psi0                 : [J][N][2]   (L, R) corner angular flux at t = 0,
                                     angle index ascending in mu
  source(step)         : [J][4]      (Q_{k,L}, Q_{k,R}, Q_{k+1/2,L}, Q_{k+1/2,R})
                                     or None for "no volumetric source"
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Callable, Optional

import numpy as np

BC_VACUUM = 0
BC_INCIDENT_ISOTROPIC = 1
BC_REFLECTING = 2

CONFIG_NAMES = {
    1: "cfg1_S4_J20_incident",
    2: "cfg2_S16_J1000_reflect_source",
    3: "cfg3_S32_J131072_thick_reflecting_shared_block",
    4: "cfg4_S128_J16384_pulse_shared_block",
    5: "cfg5_S64_J4096_heterogeneous_per_cell",
}


@dataclass
class Problem:
    cfg: int
    name: str
    n_angles: int                 # N (S_N order), even
    cells: int                    # J
    dx: np.ndarray                # [J]
    sigma_t: np.ndarray           # [J]
    sigma_s: np.ndarray           # [J]
    v: float
    dt: float
    n_steps: int
    bc_left: tuple                # (kind, value)
    bc_right: tuple               # (kind, value)
    psi0: np.ndarray              # [J][N][2]
    tol: float = 1e-10
    max_iters: int = 10_000
    _source: Optional[Callable[[int], Optional[np.ndarray]]] = field(default=None, repr=False)

    def source(self, step: int) -> Optional[np.ndarray]:
        """Q for time step `step` (0-based) as [J][4], or None when Q = 0."""
        return None if self._source is None else self._source(step)

    @property
    def unknowns(self) -> int:
        return self.cells * 4 * self.n_angles


def _const(J, val):
    return np.full(J, float(val), dtype=np.float64)


def make_problem(cfg: int, cells: Optional[int] = None, n_steps: Optional[int] = None) -> Problem:
    """Build config `cfg` (1..5).  `cells` / `n_steps` override the full size
    (used by parity tests at sizes the oracle finishes in seconds); every other
    number is the config's own."""
    if cfg == 1:
        N, J, steps = 4, 20, 5
        J = cells or J
        p = Problem(1, CONFIG_NAMES[1], N, J, _const(J, 0.5), _const(J, 1.0), _const(J, 0.5),
                    1.0, 0.1, n_steps or steps, (BC_INCIDENT_ISOTROPIC, 1.0), (BC_VACUUM, 0.0),
                    np.zeros((J, N, 2)))
        return p
    if cfg == 2:
        N, J, steps = 16, 1000, 20
        J = cells or J
        q = np.ones((J, 4), dtype=np.float64)
        return Problem(2, CONFIG_NAMES[2], N, J, _const(J, 0.1), _const(J, 1.0), _const(J, 0.9),
                       1.0, 0.05, n_steps or steps, (BC_REFLECTING, 0.0), (BC_VACUUM, 0.0),
                       np.zeros((J, N, 2)), _source=lambda step: q)
    if cfg == 3:
        N, J, steps = 32, 131072, 10
        J = cells or J
        # one draw u[j][m]; both corners get it.  The full-size draw
        # is always made so that a reduced-J problem is a prefix of the full one.
        u = np.random.default_rng(230513558).random((131072, N))[:J] if J <= 131072 else \
            np.random.default_rng(230513558).random((J, N))
        psi0 = np.repeat(u[:, :, None], 2, axis=2).copy()
        return Problem(3, CONFIG_NAMES[3], N, J, _const(J, 0.1), _const(J, 10.0), _const(J, 9.9),
                       1.0, 0.01, n_steps or steps, (BC_REFLECTING, 0.0), (BC_REFLECTING, 0.0), psi0)
    if cfg == 4:
        N, J, steps = 128, 16384, 10
        J = cells or J
        dxv = 0.2
        L = J * dxv
        j = np.arange(J, dtype=np.float64)
        xL = (j + 0.25) * dxv
        xR = (j + 0.75) * dxv
        gL = np.exp(-((xL - L / 2) / (0.1 * L)) ** 2)
        gR = np.exp(-((xR - L / 2) / (0.1 * L)) ** 2)
        q0 = np.stack([gL, gR, gL, gR], axis=1).copy()
        return Problem(4, CONFIG_NAMES[4], N, J, _const(J, dxv), _const(J, 5.0), _const(J, 4.0),
                       1.0, 0.02, n_steps or steps, (BC_INCIDENT_ISOTROPIC, 1.0), (BC_VACUUM, 0.0),
                       np.zeros((J, N, 2)), _source=lambda step: q0 if step == 0 else None)
    if cfg == 5:
        N, J, steps = 64, 4096, 10
        J = cells or J
        g = np.random.default_rng(230513560)
        Jdraw = max(J, 4096)
        sig = np.exp(g.uniform(np.log(0.1), np.log(10.0), Jdraw))
        c = g.uniform(0.5, 0.99, Jdraw)
        sig, c = sig[:J].copy(), c[:J].copy()
        q = np.ones((J, 4), dtype=np.float64)
        return Problem(5, CONFIG_NAMES[5], N, J, _const(J, 0.25), sig, c * sig,
                       1.0, 0.05, n_steps or steps, (BC_VACUUM, 0.0), (BC_VACUUM, 0.0),
                       np.zeros((J, N, 2)), _source=lambda step: q)
    raise ValueError(f"unknown config {cfg}")


def make_multi_region(cells: int = 4096, n_angles: int = 64, n_steps: int = 5) -> Problem:
    """A multi-region slab of the kind the paper times (a Reed-type problem, S64, v = 4, dt = 1, 5 steps; its
    region layout is in a figure that is not available, so the layout here is synthetic): five regions, four
    materials - a strong absorber with a strong source, a weaker absorber, a void, and two scattering regions (c = 0.9),
    one of them with a source; reflecting left, vacuum right, zero initial flux.  Region widths in units of cells/64:
    16, 8, 16, 8, 16.  A context sees 4 distinct (dx, Sigma, Sigma_s) blocks."""
    J = int(cells)
    u = J / 64.0
    edges = [0, int(16 * u), int(24 * u), int(40 * u), int(48 * u), J]
    mats = [(50.0, 0.0, 50.0), (5.0, 0.0, 0.0), (1e-12, 0.0, 0.0), (1.0, 0.9, 1.0), (1.0, 0.9, 0.0)]
    dx = _const(J, 8.0 / J)
    st, ss = np.zeros(J), np.zeros(J)
    q = np.zeros((J, 4))
    for (a, b), (sig, sigs, src) in zip(zip(edges[:-1], edges[1:]), mats):
        st[a:b], ss[a:b], q[a:b] = sig, sigs, src
    return Problem(0, f"multi_region_S{n_angles}_J{J}_reed_like", n_angles, J, dx, st, ss, 4.0, 1.0, n_steps,
                   (2, 0.0), (0, 0.0), np.zeros((J, n_angles, 2)), _source=lambda step: q)

