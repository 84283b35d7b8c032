"""The library's one entry point that allocates nothing (include/oci_static.h, csrc/phi_norm_static.cu): scalar flux and
the two stopping-rule norms with the kernel's scratch in a file-scope device array.  Collected LAST on purpose (the
suite runs with pytest -x).  The GPU test compares it with the existing workspace path on two calls in a row and passes
alone in a fresh process as well as after the other tests: nothing here depends on earlier state."""
import os
import re
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import paper_2305_13555_b200 as P  # noqa: E402
from paper_2305_13555_b200 import static_scratch as S  # noqa: E402
from workloads import make_problem  # noqa: E402


def test_static_header_symbols_are_exported_and_limits_agree():
    src = open(os.path.join(ROOT, "include", "oci_static.h")).read()
    code = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = sorted(set(re.findall(r"\b(oci_static_[a-z0-9_]+)\s*\(", code)))
    assert names == sorted(S.SYMBOLS)
    L = P.load_library()
    for nm in names:
        assert hasattr(L, nm), nm
    assert int(re.search(r"#define OCI_STATIC_MAX_CELLS (\d+)", src).group(1)) == S.MAX_CELLS
    assert S.SCRATCH_BYTES == 256 + (S.MAX_CELLS // 64) * 16 == 262400


def test_static_entry_point_source_allocates_nothing():
    src = open(os.path.join(ROOT, "paper_2305_13555_b200", "csrc", "phi_norm_static.cu")).read()
    code = re.sub(r"//.*", "", src)
    for word in ("cudaMalloc", "cudaFree", "cudaHostAlloc", "cudaMallocAsync", "cudaMallocManaged", "new ", "malloc("):
        assert word not in code, word
    assert "static __device__ __align__(256)" in code and "cudaGetSymbolAddress" in code


def _rel(a, b):
    return np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300)


@pytest.mark.gpu
def test_static_scalar_flux_norms_matches_the_workspace_path_twice():
    import torch
    p = make_problem(3, cells=5003)                      # 79 CTAs of 64 cells, the last one ragged (11 cells)
    J, N = p.cells, p.n_angles
    g = P.OCI.from_problem(p)                            # the existing path: set_flux -> phi, steps -> phi
    _, w = g.get_quadrature()
    S.static_prepare()
    w_d = torch.from_numpy(w).cuda()
    psi_d = torch.empty((J, N, 4), dtype=torch.float64, device="cuda")
    phi_d = [torch.full((J, 4), -7.0, dtype=torch.float64, device="cuda") for _ in range(2)]
    norms_d = torch.full((2,), -1.0, dtype=torch.float64, device="cuda")

    # call 1: the initial condition; no phi_old -> d = 0
    phi_ref0 = g.get_scalar_flux()
    g.get_angular_flux_dev(psi_d)
    S.static_scalar_flux_norms(psi_d, w_d, None, phi_d[0], norms_d)
    torch.cuda.synchronize()
    out0, nrm0 = phi_d[0].cpu().numpy(), norms_d.cpu().numpy()
    assert _rel(out0, phi_ref0) < 1e-12
    assert nrm0[0] == 0.0 and abs(nrm0[1] - np.max(np.abs(phi_ref0))) <= 1e-12 * np.max(np.abs(phi_ref0))

    # call 2, right behind it on the same stream: the state after two iterations of a time step, against the previous phi
    g.set_source(p.source(0))
    g.oci_step(-1.0, 2)
    phi_ref1 = g.get_scalar_flux()
    g.get_angular_flux_dev(psi_d)
    S.static_scalar_flux_norms(psi_d, w_d, phi_d[0], phi_d[1], norms_d)
    S.static_scalar_flux_norms(psi_d, w_d, phi_d[0], phi_d[1], norms_d)       # and once more: same inputs, same outputs
    torch.cuda.synchronize()
    out1, nrm1 = phi_d[1].cpu().numpy(), norms_d.cpu().numpy()
    assert _rel(out1, phi_ref1) < 1e-12
    d_ref, r_ref = np.max(np.abs(phi_ref1 - phi_ref0)), np.max(np.abs(phi_ref1))
    assert d_ref > 0.0
    assert abs(nrm1[0] - d_ref) <= 1e-12 * r_ref and abs(nrm1[1] - r_ref) <= 1e-12 * r_ref
    g.close()

    # a small and a one-cell problem reuse the same scratch array (stale pairs of the larger call must not be read)
    for cells in (1, 130):
        q = make_problem(2, cells=cells)
        h = P.OCI.from_problem(q)
        _, wq = h.get_quadrature()
        ps = torch.empty((cells, q.n_angles, 4), dtype=torch.float64, device="cuda")
        h.get_angular_flux_dev(ps)
        ph = torch.empty((cells, 4), dtype=torch.float64, device="cuda")
        S.static_scalar_flux_norms(ps, torch.from_numpy(wq).cuda(), None, ph, norms_d)
        torch.cuda.synchronize()
        ref = h.get_scalar_flux()
        assert _rel(ph.cpu().numpy(), ref) < 1e-12
        assert abs(norms_d.cpu().numpy()[1] - np.max(np.abs(ref))) <= 1e-12 * np.max(np.abs(ref))
        h.close()


@pytest.mark.gpu
def test_static_entry_point_rejects_sizes_beyond_its_scratch():
    import torch
    t = torch.zeros(64, dtype=torch.float64, device="cuda")
    for cells, n_angles in ((S.MAX_CELLS + 1, 4), (0, 4), (10, 3), (10, 514)):
        with pytest.raises(P.OCIError) as e:
            S.static_scalar_flux_norms(t, t, None, t, t, cells=cells, n_angles=n_angles)
        assert e.value.code == -1 and "oci_static_scalar_flux_norms" in str(e.value)
    with pytest.raises(P.OCIError):
        S.static_scalar_flux_norms(t, t, t, t, t, cells=1, n_angles=2)        # phi_old aliases phi
