"""Whole-problem dense MB-SCB system, assembled in the TEST directly from the
balance equations (4)-(7) with the closures (8)-(11) of PAPER.md:74-96, and
solved with numpy.  This is the paper's own statement that a whole-problem
linear solve "will produce the same solutions ... as implementations that
manually conduct a sweep or a cell inversion", used as a
brute-force pin for the oracle.  It deliberately does NOT go through the 4x4 /
4Nx4N matrices of eqs. (13)-(28): every term is added equation by equation
through a generic "edge flux" closure, so a wrong entry, sign or index in the
oracle's A+-, b+-, c+-, S shows up as a mismatch.

Unknown numbering here is this file's own: u(j, m, t, side), t in {0: time
average k, 1: time edge k+1/2}, side in {0: L, 1: R}.
"""
import numpy as np

VAC, INC, REF = 0, 1, 2


def solve_step(dx, sig, sigs, v, dt, mu, w, bcL, bcR, psi_prev, Q):
    """One converged time step.  psi_prev [J][N][2], Q [J][4] (k,L),(k,R),(k+1/2,L),(k+1/2,R).
    Returns psi [J][N][2(t)][2(side)]."""
    J, N = len(dx), len(mu)

    def u(j, m, t, side):
        return ((j * N + m) * 2 + t) * 2 + side

    M = np.zeros((J * N * 4, J * N * 4))
    rhs = np.zeros(J * N * 4)

    def add_edge(row, coef, j_face, m, t):
        """add coef * psi_{m,t,face} where face index j_face means x_{j_face-1/2}
        (j_face = 0 .. J), using the upstream prescription (10),(11)."""
        if mu[m] > 0:
            if j_face > 0:
                M[row, u(j_face - 1, m, t, 1)] += coef          # psi_{j-1,R}
            else:                                               # left boundary
                kind, val = bcL
                if kind == INC:
                    rhs[row] -= coef * val
                elif kind == REF:
                    M[row, u(0, N - 1 - m, t, 0)] += coef       # mirror angle leaving at x=0
        else:
            if j_face < J:
                M[row, u(j_face, m, t, 0)] += coef              # psi_{j,L}
            else:
                kind, val = bcR
                if kind == INC:
                    rhs[row] -= coef * val
                elif kind == REF:
                    M[row, u(J - 1, N - 1 - m, t, 1)] += coef

    for j in range(J):
        h = dx[j]
        for m in range(N):
            for t in (0, 1):
                for side in (0, 1):
                    row = u(j, m, t, side)
                    # --- time-derivative term
                    if t == 0:      # eqs (4),(5): (h/2)(1/v)(psi_{k+1/2} - psi_{k-1/2})/dt
                        M[row, u(j, m, 1, side)] += h / 2 / v / dt
                        rhs[row] += h / 2 / v / dt * psi_prev[j, m, side]
                    else:           # eqs (6),(7): (h/2)(1/v)(psi_{k+1/2} - psi_k)/(dt/2)
                        M[row, u(j, m, 1, side)] += h / 2 / v / (dt / 2)
                        M[row, u(j, m, 0, side)] -= h / 2 / v / (dt / 2)
                    # --- streaming term with the midpoint closure (8),(9)
                    if side == 0:   # mu [ (L+R)/2 - psi_{j-1/2} ]
                        M[row, u(j, m, t, 0)] += mu[m] / 2
                        M[row, u(j, m, t, 1)] += mu[m] / 2
                        add_edge(row, -mu[m], j, m, t)
                    else:           # mu [ psi_{j+1/2} - (L+R)/2 ]
                        M[row, u(j, m, t, 0)] -= mu[m] / 2
                        M[row, u(j, m, t, 1)] -= mu[m] / 2
                        add_edge(row, +mu[m], j + 1, m, t)
                    # --- collision
                    M[row, u(j, m, t, side)] += h / 2 * sig[j]
                    # --- isotropic scattering + source, (h/2)(1/2)(Sigma_s phi + Q)
                    for nn in range(N):
                        M[row, u(j, nn, t, side)] -= h / 2 / 2 * sigs[j] * w[nn]
                    rhs[row] += h / 2 / 2 * Q[j, 2 * t + side]
    x = np.linalg.solve(M, rhs)
    return x.reshape(J, N, 2, 2)


def to_slots(psi):
    """[J][N][t][side] -> the oracle's [J][N][4] slot order (k,L),(k,R),(k+1/2,L),(k+1/2,R)."""
    J, N = psi.shape[:2]
    return psi.reshape(J, N, 4)
