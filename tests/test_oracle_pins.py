"""Pins for the CPU oracle against what the paper and the mathematics fix.
Each test names the passage it pins (P:<line> = /root/reference/PAPER.md line).
None of these compares the oracle with itself or with the CUDA path."""
import numpy as np
import pytest

from oracle import A4, Oracle, cell_matrix, gauss_legendre, lu_factor, lu_solve
from tests import brute_force as bf

VAC, INC, REF = 0, 1, 2


# ----------------------------------------------------------------- quadrature (eq. 1)
@pytest.mark.parametrize("N", [2, 4, 8, 16, 32, 64, 128, 256])
def test_quadrature_identities_and_library(N):
    mu, w = gauss_legendre(N)
    assert np.all(np.diff(mu) > 0)                      # ascending
    assert abs(w.sum() - 2.0) < 1e-13
    assert abs((w * mu).sum()) < 1e-14
    assert abs((w * mu**2).sum() - 2.0 / 3.0) < 1e-13
    assert np.max(np.abs(mu + mu[::-1])) < 1e-15        # mu_m = -mu_{N-1-m}
    assert np.max(np.abs(w - w[::-1])) < 1e-14
    x, ww = np.polynomial.legendre.leggauss(N)          # library routine
    assert np.max(np.abs(mu - x)) < 5e-15
    assert np.max(np.abs(w - ww)) < 5e-14
    # exact for polynomials of degree <= 2N-1
    for deg in (2 * N - 2, 2 * N - 1):
        exact = 0.0 if deg % 2 else 2.0 / (deg + 1)
        assert abs((w * mu**deg).sum() - exact) < 1e-13


# ----------------------------------------------------------------- dense LU (P:208 `gesv`)
def test_lu_matches_numpy_with_pivoting():
    rng = np.random.default_rng(7)
    for n in (1, 4, 16, 33):
        A = rng.standard_normal((n, n))
        A[0, 0] = 1e-14                                 # forces a row interchange
        b = rng.standard_normal(n)
        LU, piv, info = lu_factor(A)
        assert info == 0
        if n > 1:
            assert piv[0] != 0
        x = lu_solve(LU, piv, b)
        assert np.allclose(x, np.linalg.solve(A, b), rtol=1e-10, atol=1e-12)
    _, _, info = lu_factor(np.zeros((3, 3)))
    assert info != 0                                    # singular is reported


# ----------------------------------------------------------------- A+-, S (eqs 13,16,20-22)
def test_cell_matrix_inverse_bruteforce_and_woodbury():
    """B = A - S at S2/S4/S8: B^{-1} via the oracle's LU against numpy's inverse, and against the
    Woodbury form (S has rank 4), an independent algebraic route."""
    for N, dx, sig, sigs, v, dt in [(2, 0.5, 1.0, 0.5, 1.0, 0.1), (4, 0.1, 10.0, 9.9, 1.0, 0.01),
                                    (8, 0.25, 0.3, 0.29, 2.0, 5.0)]:
        mu, w = gauss_legendre(N)
        B = cell_matrix(mu, w, dx, sig, sigs, v, dt)
        n = 4 * N
        LU, piv, info = lu_factor(B)
        assert info == 0
        Binv = np.column_stack([lu_solve(LU, piv, e) for e in np.eye(n)])
        assert np.max(np.abs(B @ Binv - np.eye(n))) < 1e-13
        assert np.max(np.abs(Binv - np.linalg.inv(B))) < 1e-12 * np.max(np.abs(Binv))
        # Woodbury: A block diagonal, S = U V with U = (dx sigs/4)(1_N (x) I4), V = w^T (x) I4
        A = np.zeros((n, n))
        for m in range(N):
            A[4 * m:4 * m + 4, 4 * m:4 * m + 4] = A4(mu[m], dx, sig, v, dt)
        U = dx * sigs / 4 * np.kron(np.ones((N, 1)), np.eye(4))
        V = np.kron(w[None, :], np.eye(4))
        assert np.max(np.abs(A - U @ V - B)) < 1e-15
        Ai = np.linalg.inv(A)
        Wb = Ai + Ai @ U @ np.linalg.inv(np.eye(4) - V @ Ai @ U) @ V @ Ai
        assert np.max(np.abs(Wb - Binv)) < 1e-12 * np.max(np.abs(Binv))


def test_A4_from_balance_equations():
    """The 4x4 of eqs (13),(16) (rows repaired, readings G1-G3) must equal the Jacobian of the
    residuals of eqs (4)-(7) with the closures (8)-(11), formed here by finite differencing the
    equations as printed (they are linear, so the difference is exact up to rounding)."""
    dx, sig, v, dt = 0.37, 1.9, 1.3, 0.21

    def residual(x, mu):
        kL, kR, hL, hR = x          # psi_{k,L}, psi_{k,R}, psi_{k+1/2,L}, psi_{k+1/2,R}
        up_k = up_h = 0.0           # neighbour / previous-step data set to zero
        if mu > 0:
            eL_k, eR_k, eL_h, eR_h = up_k, kR, up_h, hR
        else:
            eL_k, eR_k, eL_h, eR_h = kL, up_k, hL, up_h
        r4 = dx / 2 / v * (hL - 0.0) / dt + mu * ((kL + kR) / 2 - eL_k) + dx / 2 * sig * kL
        r5 = dx / 2 / v * (hR - 0.0) / dt + mu * (eR_k - (kL + kR) / 2) + dx / 2 * sig * kR
        r6 = dx / 2 / v * (hL - kL) / (dt / 2) + mu * ((hL + hR) / 2 - eL_h) + dx / 2 * sig * hL
        r7 = dx / 2 / v * (hR - kR) / (dt / 2) + mu * (eR_h - (hL + hR) / 2) + dx / 2 * sig * hR
        return np.array([r4, r5, r6, r7])

    for mu in (0.83, -0.83, 0.05, -0.31):
        Jac = np.column_stack([residual(e, mu) for e in np.eye(4)])
        assert np.max(np.abs(Jac - A4(mu, dx, sig, v, dt))) < 1e-15


# ----------------------------------------------------------------- brute force whole problem
def _run(o, scheme, steps, q=None, tol=1e-13, max_iters=200_000):
    o.set_source(q)
    for _ in range(steps):
        st, it, _ = (o.oci_step if scheme == "oci" else o.si_step)(tol, max_iters)
        assert st == 0
    return o.angular_flux()


@pytest.mark.parametrize("bcL,bcR", [((VAC, 0.0), (VAC, 0.0)), ((INC, 1.0), (VAC, 0.0)),
                                     ((REF, 0.0), (INC, 0.7)), ((REF, 0.0), (REF, 0.0)),
                                     ((VAC, 0.0), (REF, 0.0))])
@pytest.mark.parametrize("N", [2, 4])
def test_converged_step_equals_whole_problem_solve(N, bcL, bcR):
    """Eqs (12)-(28) iterated to convergence == eqs (4)-(11) solved as one dense system.
    Heterogeneous cells, nonzero IC, all four Q slots different, two consecutive steps."""
    rng = np.random.default_rng(100 + N)
    J = 5
    dx = rng.uniform(0.2, 0.9, J)
    sig = rng.uniform(0.5, 3.0, J)
    sigs = sig * rng.uniform(0.2, 0.9, J)
    v, dt = 1.7, 0.23
    psi0 = rng.uniform(0.0, 1.0, (J, N, 2))
    Q = rng.uniform(0.0, 1.0, (J, 4))
    mu, w = np.polynomial.legendre.leggauss(N)
    prev = psi0
    ref_steps = []
    for _ in range(2):
        x = bf.solve_step(dx, sig, sigs, v, dt, mu, w, bcL, bcR, prev, Q)
        ref_steps.append(bf.to_slots(x))
        prev = x[:, :, 1, :]
    for scheme in ("oci", "si"):
        o = Oracle(dx, sig, sigs, v, dt, N, bcL, bcR)
        o.setup()
        o.set_flux(psi0)
        o.set_source(Q)
        for k in range(2):
            st, it, res = (o.oci_step if scheme == "oci" else o.si_step)(1e-14, 100_000)
            assert st == 0
            got = o.angular_flux()
            assert np.max(np.abs(got - ref_steps[k])) < 2e-11 * np.max(np.abs(ref_steps[k])), scheme


# ----------------------------------------------------------------- MB closed form (eqs 2,3)
@pytest.mark.parametrize("scheme", ["oci", "si"])
def test_zero_dimensional_decay_closed_form(scheme):
    """Reflecting both sides, flat isotropic IC psi=1, Q=0: every psi_{k+1/2} = 1/(1+z+z^2/2) of the
    previous edge value and psi_k = (1+z/2)/(1+z+z^2/2), z = (Sigma-Sigma_s) v dt (eqs. 2,3)."""
    sig, sigs, v, dt, N, J = 2.0, 1.2, 1.5, 0.07, 4, 6
    z = (sig - sigs) * v * dt
    g = 1.0 / (1.0 + z + z * z / 2.0)
    o = Oracle(np.full(J, 0.3), np.full(J, sig), np.full(J, sigs), v, dt, N, (REF, 0), (REF, 0))
    o.setup()
    o.set_flux(np.ones((J, N, 2)))
    edge = 1.0
    for _ in range(3):
        st, _, _ = (o.oci_step if scheme == "oci" else o.si_step)(1e-14, 100_000)
        assert st == 0
        psi = o.angular_flux()
        assert np.max(np.abs(psi[:, :, 2:] - edge * g)) < 1e-11
        assert np.max(np.abs(psi[:, :, :2] - edge * g * (1 + z / 2))) < 1e-11
        edge *= g
    assert abs(g - 0.9195165549760558) < 1e-15          # value of the closed form itself


# ----------------------------------------------------------------- SCB closed form (eqs 4-11)
@pytest.mark.parametrize("scheme", ["oci", "si"])
def test_steady_pure_absorber_attenuation_closed_form(scheme):
    """dt -> infinity, Sigma_s = 0, incident 1 on the left, vacuum right: the SCB outgoing corner
    flux is (1/(1+tau+tau^2/2))^(j+1), tau = Sigma dx/mu_m, for mu_m > 0 and 0 for mu_m < 0."""
    N, J, dx, sig = 4, 7, 0.8, 1.3
    o = Oracle(np.full(J, dx), np.full(J, sig), np.zeros(J), 1.0, 1e12, N, (INC, 1.0), (VAC, 0.0))
    o.setup()
    o.set_flux(np.zeros((J, N, 2)))
    st, it, _ = (o.oci_step if scheme == "oci" else o.si_step)(1e-15, 1000)
    assert st == 0
    mu, _ = o.quadrature()
    psi = o.angular_flux()
    j = np.arange(J)
    for m in range(N):
        if mu[m] > 0:
            tau = sig * dx / mu[m]
            exact = (1.0 / (1.0 + tau + tau * tau / 2.0)) ** (j + 1)
            assert np.max(np.abs(psi[:, m, 1] - exact)) < 1e-10
            assert np.max(np.abs(psi[:, m, 3] - exact)) < 1e-10
        else:
            assert np.max(np.abs(psi[:, m, :])) == 0.0
    tau = 1.3 * 0.8 / np.polynomial.legendre.leggauss(2)[0][1]
    assert abs(1 / (1 + tau + tau * tau / 2) - 0.2260534341013726) < 1e-15


def test_pure_absorber_converges_to_exponential_second_order():
    """P:210 verification problem; north_star: exp(-Sigma x/mu) in the fine-mesh limit.  After the
    front has passed, psi_m(x_{j+1/2}) -> exp(-Sigma x/mu_m); halving dx cuts the error ~4x."""
    sig, X, N, v = 1.0, 2.0, 4, 1.0
    errs = []
    for J in (20, 40, 80):
        dx = X / J
        o = Oracle(np.full(J, dx), np.full(J, sig), np.zeros(J), v, 0.5, N, (INC, 1.0), (VAC, 0.0))
        o.setup()
        o.set_flux(np.zeros((J, N, 2)))
        for _ in range(120):                             # t = 60 >> X/(v min mu+) = 5.9
            st, _, _ = o.oci_step(1e-13, 100_000)
            assert st == 0
        mu, _ = o.quadrature()
        psi = o.angular_flux()
        x = (np.arange(J) + 1) * dx
        e = 0.0
        for m in range(N):
            if mu[m] > 0:
                e = max(e, np.max(np.abs(psi[:, m, 3] - np.exp(-sig * x / mu[m]))))
        errs.append(e)
    assert errs[0] < 1e-2 and errs[2] < 5e-4
    assert 3.5 < errs[0] / errs[1] < 4.5
    assert 3.5 < errs[1] / errs[2] < 4.5


@pytest.mark.parametrize("scheme", ["oci", "si"])
def test_steady_infinite_medium_source(scheme):
    """Reflecting both sides, dt -> infinity: phi = Q/(Sigma - Sigma_s) in all four slots."""
    N, J, sig, sigs, Q = 4, 4, 1.0, 0.6, 0.35
    o = Oracle(np.full(J, 2.0), np.full(J, sig), np.full(J, sigs), 1.0, 1e12, N, (REF, 0), (REF, 0))
    o.setup()
    o.set_flux(np.zeros((J, N, 2)))
    o.set_source(np.full((J, 4), Q))
    st, it, _ = (o.oci_step if scheme == "oci" else o.si_step)(1e-14, 100_000)
    assert st == 0
    assert np.max(np.abs(o.scalar_flux() - Q / (sig - sigs))) < 1e-10


# ----------------------------------------------------------------- particle balance (eqs 4-7 summed)
def test_particle_balance_every_oci_iterate_and_converged():
    """sum_m w_m [(4)+(5)] and [(6)+(7)]: per cell, with the inflow taken from the previous iterate,
    balance closes at EVERY OCI iterate; with the converged inflow it closes for SI too."""
    rng = np.random.default_rng(11)
    N, J, v, dt = 4, 9, 1.3, 0.4
    dx = rng.uniform(0.2, 1.0, J)
    sig = rng.uniform(0.5, 2.0, J)
    sigs = sig * rng.uniform(0.1, 0.95, J)
    Q = rng.uniform(0, 1, (J, 4))
    psi0 = rng.uniform(0, 1, (J, N, 2))
    bcL, bcR = (INC, 0.8), (VAC, 0.0)
    gam = 1.0 / (v * dt)

    def check(psi_new, psi_lag, prev, tol):
        mu, w = np.polynomial.legendre.leggauss(N)
        phi = np.einsum("m,jms->js", w, psi_new)
        phi_prev = np.einsum("m,jms->js", w, prev)
        for j in range(J):
            for t in (0, 1):                         # k and k+1/2 balance
                Jout = Jin = 0.0
                for m in range(N):
                    if mu[m] > 0:
                        out = psi_new[j, m, 2 * t + 1]
                        inc = psi_lag[j - 1, m, 2 * t + 1] if j > 0 else bcL[1]
                    else:
                        out = psi_new[j, m, 2 * t + 0]
                        inc = psi_lag[j + 1, m, 2 * t + 0] if j < J - 1 else 0.0
                    Jout += w[m] * abs(mu[m]) * out
                    Jin += w[m] * abs(mu[m]) * inc
                h = dx[j]
                if t == 0:
                    ddt = gam * h / 2 * ((phi[j, 2] - phi_prev[j, 0]) + (phi[j, 3] - phi_prev[j, 1]))
                else:
                    ddt = 2 * gam * h / 2 * ((phi[j, 2] - phi[j, 0]) + (phi[j, 3] - phi[j, 1]))
                absorb = h / 2 * (sig[j] - sigs[j]) * (phi[j, 2 * t] + phi[j, 2 * t + 1])
                src = h / 2 * (Q[j, 2 * t] + Q[j, 2 * t + 1])
                scale = abs(ddt) + Jout + Jin + absorb + src
                assert abs(ddt + Jout - Jin + absorb - src) < tol * scale

    o = Oracle(dx, sig, sigs, v, dt, N, bcL, bcR)
    o.setup()
    o.set_flux(psi0)
    o.set_source(Q)
    prev = psi0
    lag = o.angular_flux()
    for _ in range(6):                               # every iterate
        o.oci_iteration()
        new = o.angular_flux()
        check(new, lag, prev, 1e-13)
        lag = new
    for scheme in ("oci", "si"):                     # converged: inflow = own solution
        o = Oracle(dx, sig, sigs, v, dt, N, bcL, bcR)
        o.setup()
        o.set_flux(psi0)
        o.set_source(Q)
        st, _, _ = (o.oci_step if scheme == "oci" else o.si_step)(1e-14, 100_000)
        assert st == 0
        x = o.angular_flux()
        check(x, x, prev, 1e-11)
        assert np.array_equal(o.prev_edge_flux(), x[:, :, 2:])     # commit


# ----------------------------------------------------------------- OCI == SI
@pytest.mark.parametrize("cfg,cells,steps", [(1, 20, 5), (2, 120, 3), (3, 96, 2), (4, 24, 2), (5, 48, 2)])
def test_oci_and_si_agree_on_configs(cfg, cells, steps):
    from workloads import make_problem
    p = make_problem(cfg, cells=cells, n_steps=steps)
    a, b = Oracle.from_problem(p, threads=4), Oracle.from_problem(p, threads=4)
    for k in range(steps):
        a.set_source(p.source(k))
        b.set_source(p.source(k))
        sa, ia, _ = a.oci_step(p.tol, p.max_iters)
        sb, ib, _ = b.si_step(p.tol, p.max_iters)
        assert sa == 0 and sb == 0
    fa, fb = a.scalar_flux(), b.scalar_flux()
    assert np.max(np.abs(fa - fb)) < 1e-8 * np.max(np.abs(fa))
    pa, pb = a.angular_flux(), b.angular_flux()
    assert np.max(np.abs(pa - pb)) < 1e-8 * np.max(np.abs(pa))


def test_threads_do_not_change_results():
    from workloads import make_problem
    p = make_problem(5, cells=40, n_steps=1)
    outs = []
    for th in (1, 4):
        for scheme in ("oci", "si"):
            o = Oracle.from_problem(p, threads=th)
            o.set_source(p.source(0))
            (o.oci_step if scheme == "oci" else o.si_step)(-1.0, 4)
            outs.append(o.angular_flux())
    assert np.array_equal(outs[0], outs[2]) and np.array_equal(outs[1], outs[3])


# ----------------------------------------------------------------- spectral radii (Fig. 1)
def _rho(o, scheme, J, N, iters=400, skip=200, seed=3):
    """Power iteration on the homogeneous problem (Q = 0, psi_{k-1/2} = 0): the iterate IS the error."""
    rng = np.random.default_rng(seed)
    o.set_flux(np.zeros((J, N, 2)))
    o.set_source(None)
    o.set_iterate(rng.uniform(0.5, 1.5, (J, 4 * N)))
    f = o.oci_iteration if scheme == "oci" else o.si_iteration
    ds = []
    for _ in range(iters):
        d, r = f()
        ds.append(d)
    ds = np.array(ds)
    return (ds[-1] / ds[skip]) ** (1.0 / (iters - 1 - skip))


def test_si_spectral_radius_infinite_medium():
    """Steady (dt->inf) thick slab: rho_SI -> c = Sigma_s/Sigma ("depends strongly on the
    scattering ratio ... nearly independent of cell optical thickness")."""
    N, J, c = 4, 60, 0.9
    for dxv in (1.0, 2.0):
        o = Oracle(np.full(J, dxv), np.ones(J), np.full(J, c), 1.0, 1e12, N, (REF, 0), (REF, 0))
        o.setup()
        rho = _rho(o, "si", J, N, iters=300, skip=150)
        assert abs(rho - c) < 0.01 * c


def test_si_spectral_radius_time_dependent_effective_ratio():
    """With a finite dt the flat-mode SI error obeys [[S, g],[-2g, S+2g]] E' = Sigma_s E (eqs. 2,3,
    g = 1/(v dt)): eigenvalues Sigma_s/((S+g) +- i g), modulus Sigma_s/sqrt((S+g)^2+g^2) (reading
    S12); the backward-Euler-like Sigma_s/(S+g) quoted in north_star is an upper bound."""
    N, J, sig, sigs, v, dt = 4, 48, 1.0, 0.9, 1.0, 1.0
    g = 1.0 / (v * dt)
    mb = sigs / np.sqrt((sig + g) ** 2 + g**2)
    be = sigs / (sig + g)
    # thick (48 mfp) vacuum/vacuum slab: the interior flat mode dominates.  (Lagged reflecting
    # boundaries, reading S4, add a boundary mode slightly ABOVE the infinite-medium value, so the
    # infinite medium is approached from a thick finite slab here.)
    o = Oracle(np.full(J, 1.0), np.full(J, sig), np.full(J, sigs), v, dt, N, (VAC, 0), (VAC, 0))
    o.setup()
    rho = _rho(o, "si", J, N, iters=200, skip=100)
    assert abs(rho - mb) < 0.02 * mb
    assert rho < be * 0.95


def test_oci_spectral_radius_falls_with_cell_thickness():
    """rho_OCI decreases substantially as the cell optical thickness grows (steady S4,
    c = 0.99, reflecting)."""
    N, J = 4, 24
    rhos = []
    for thick in (0.05, 0.5, 5.0):
        o = Oracle(np.full(J, thick), np.ones(J), np.full(J, 0.99), 1.0, 1e12, N, (REF, 0), (REF, 0))
        o.setup()
        rhos.append(_rho(o, "oci", J, N, iters=1500, skip=700))
    assert rhos[0] > rhos[1] > rhos[2]
    assert rhos[0] > 0.99 and rhos[2] < 0.95
    # and OCI needs more iterations than SI on thin cells
    o = Oracle(np.full(J, 0.05), np.ones(J), np.full(J, 0.5), 1.0, 1e12, N, (REF, 0), (REF, 0))
    o.setup()
    r_oci = _rho(o, "oci", J, N, iters=600, skip=300)
    r_si = _rho(o, "si", J, N, iters=60, skip=20)
    assert r_oci > r_si


# ----------------------------------------------------------------- stopping rule / API behaviour
def test_fixed_iteration_mode_and_status():
    from workloads import make_problem
    p = make_problem(1)
    o = Oracle.from_problem(p)
    st, it, _ = o.oci_step(-1.0, 5)
    assert (st, it) == (1, 5)                              # tol<0: exactly max_iters, NOT_CONVERGED
    o = Oracle.from_problem(p)
    st, it, res = o.oci_step(1e-10, 10_000)
    assert st == 0 and res <= 1e-10
    # all-zero problem converges at the first iteration (d = r = 0)
    z = Oracle(np.ones(3), np.ones(3), np.zeros(3), 1.0, 1.0, 2)
    z.setup()
    z.set_flux(np.zeros((3, 2, 2)))
    assert z.oci_step(1e-10, 100)[:2] == (0, 1)
    assert z.si_step(1e-10, 100)[:2] == (0, 1)
    with pytest.raises(ValueError):
        Oracle(np.ones(3), np.ones(3), np.zeros(3), 1.0, 1.0, 3)   # odd N
    with pytest.raises(ValueError):
        Oracle(-np.ones(3), np.ones(3), np.zeros(3), 1.0, 1.0, 2)  # dx <= 0


# ----------------------------------------------------------------- stopping-rule arithmetic (reading S2)
def _norm_problem(scheme_seed=0):
    """Small heterogeneous slab whose source is concentrated in the k slots (0, 1) of one interior cell, so
    that both max-norms of the first iterations sit in a k slot of an interior cell: a reduction over the
    wrong slot range (k+1/2 only), over a sub-range of cells, or over phi_old instead of phi_new would miss it."""
    rng = np.random.default_rng(2305 + scheme_seed)
    N, J, v, dt = 4, 11, 1.1, 0.6
    dx = rng.uniform(0.3, 0.9, J)
    sig = rng.uniform(0.6, 2.5, J)
    sigs = sig * rng.uniform(0.3, 0.9, J)
    Q = np.full((J, 4), 1e-3)
    Q[6, 0], Q[6, 1] = 40.0, 55.0                     # interior cell 6, slots (k,L), (k,R)
    psi0 = rng.uniform(0.0, 0.05, (J, N, 2))
    o = Oracle(dx, sig, sigs, v, dt, N, (INC, 0.3), (REF, 0.0))
    o.setup()
    o.set_flux(psi0)
    o.set_source(Q)
    return o, N, J


@pytest.mark.parametrize("scheme", ["oci", "si"])
def test_returned_norms_equal_their_definition(scheme):
    """Reading S2 ("ceases changing"; north_star "tolerance on scalar flux"): after
    an iteration d = max_{j,s}|phi^(l+1) - phi^(l)| and r = max_{j,s}|phi^(l+1)| over ALL cells and ALL four
    slots, phi = sum_m w_m psi_m (eq. 18).  phi is re-formed here from the angular fluxes with
    numpy.einsum and numpy's Gauss-Legendre weights, before and after each of several iterations."""
    o, N, J = _norm_problem(0 if scheme == "oci" else 1)
    _, w = np.polynomial.legendre.leggauss(N)
    f = o.oci_iteration if scheme == "oci" else o.si_iteration
    phi_old = np.einsum("m,jms->js", w, o.angular_flux())
    seen_k_slot_interior = False
    for it in range(6):
        d, r = f()
        phi_new = np.einsum("m,jms->js", w, o.angular_flux())
        d_np, r_np = np.max(np.abs(phi_new - phi_old)), np.max(np.abs(phi_new))
        assert abs(d - d_np) <= 4e-15 * r_np, (it, d, d_np)
        assert abs(r - r_np) <= 4e-15 * r_np, (it, r, r_np)
        assert np.max(np.abs(o.scalar_flux() - phi_new)) <= 4e-15 * r_np          # eq. (18) itself
        jd, sd = np.unravel_index(np.argmax(np.abs(phi_new - phi_old)), phi_new.shape)
        jr, sr = np.unravel_index(np.argmax(np.abs(phi_new)), phi_new.shape)
        if it == 0:
            # the construction works: both maxima in a k slot (0/1) of the interior cell
            assert (jd, jr) == (6, 6) and sd in (0, 1) and sr in (0, 1)
            seen_k_slot_interior = True
            # ... and restricting either reduction to the k+1/2 slots, to the edge cells, or taking
            # max|phi_old| for r would give a different number (so the pin can fail)
            assert np.max(np.abs(phi_new[:, 2:] - phi_old[:, 2:])) < 0.9 * d
            assert np.max(np.abs(phi_new[[0, -1]])) < 0.9 * r
            assert np.max(np.abs(phi_old)) < 0.9 * r
        phi_old = phi_new
    assert seen_k_slot_interior


@pytest.mark.parametrize("scheme", ["oci", "si"])
def test_converged_branches(scheme):
    """The three branches of the stopping rule (reading S2): tol < 0 never converges; r = 0 converges iff
    d = 0; otherwise converged iff d <= tol * r, with equality counting (the boundary is found with
    nextafter, so '<' instead of '<=' or a test against the previous r fails)."""
    def fresh():
        return _norm_problem(7)[0]

    step = (lambda o, tol, mx: o.oci_step(tol, mx)) if scheme == "oci" else (lambda o, tol, mx: o.si_step(tol, mx))
    o = fresh()
    d, r = (o.oci_iteration if scheme == "oci" else o.si_iteration)()
    assert d > 0 and r > 0
    # smallest tol with tol * r >= d
    t = d / r
    while t * r < d:
        t = np.nextafter(t, np.inf)
    while np.nextafter(t, 0.0) * r >= d:
        t = np.nextafter(t, 0.0)
    st, it, res = step(fresh(), t, 50)
    assert (st, it) == (0, 1) and res == d / r                       # d <= tol r holds with equality or by one ulp
    st, it, _ = step(fresh(), np.nextafter(t, 0.0), 50)
    assert it > 1                                                    # one ulp below: the first iterate is not accepted
    # tol < 0: never, whatever d and r are; status 1 and exactly max_iters iterations
    assert step(fresh(), -1.0, 4)[:2] == (1, 4)
    assert step(fresh(), -0.0, 3)[0] in (0, 1)                       # -0.0 >= 0 is true: behaves as tol = 0
    # tol = 0: converged only when the iterate stops changing bit for bit
    o = fresh()
    st, it, res = step(o, 0.0, 100_000)
    assert st == 0 and res == 0.0 and it > 10                        # d == 0 exactly, reached only after many iterations
    # r = 0 and d = 0 (all-zero problem): converged at the first iteration, resid = d = 0
    z = Oracle(np.ones(3), np.ones(3), np.full(3, 0.5), 1.0, 1.0, 2)
    z.setup()
    z.set_flux(np.zeros((3, 2, 2)))
    assert step(z, 1e-10, 100) == (0, 1, 0.0)
    # r = 0 at tol = 0 as well (0 <= 0 * 0)
    z.set_flux(np.zeros((3, 2, 2)))
    assert step(z, 0.0, 100)[:2] == (0, 1)


# ----------------------------------------------------------------- Fig. 1-style map, row f4's second half
def test_rho_map_trends_and_stored_table():
    """`python -m oracle.rho_map` (steady S4, reflecting): what P:31 and P:37 state must hold over the whole grid -
    rho_OCI falls monotonically as the cell optical thickness grows, rho_SI "depends strongly on the scattering ratio
    and is nearly independent of cell optical thickness" (within a few per cent of c once cells are >= 0.5 mfp), OCI
    loses to SI on thin cells and wins on thick ones - and the committed table is what the script writes."""
    import os
    from oracle import rho_map
    txt, grid = rho_map.table(24)
    for c in rho_map.CS:
        oci = [grid[(th, c)][0] for th in rho_map.THICK]
        assert all(a > b for a, b in zip(oci, oci[1:])), (c, oci)
        for th in rho_map.THICK:
            if th >= 0.5:
                assert abs(grid[(th, c)][1] - c) < 0.09 * c, (th, c, grid[(th, c)])
        assert grid[(0.05, c)][0] > grid[(0.05, c)][1] and grid[(10.0, c)][0] < grid[(10.0, c)][1]
    stored = open(os.path.join(os.path.dirname(rho_map.__file__), "rho_map_S4.txt")).read()
    assert stored == txt
