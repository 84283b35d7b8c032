"""Host-side checks that need no GPU: the C-ABI library builds, loads and exports every symbol that
include/oci.h declares; the host-only entry points (oci_create validation, quadrature, block
classification, workspace sizing, call-order errors) behave as the header states; and the binding
fails loudly, with no CPU fallback, when there is no CUDA device."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import paper_2305_13555_b200 as P

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "oci.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"\b((?:oci|si)_[a-z0-9_]+)\s*\(", src)
    return sorted(set(names))


def test_library_exports_every_declared_symbol():
    L = P.load_library()
    names = declared_symbols()
    assert "oci_create" in names and "oci_setup" in names and "oci_step" in names and "si_step" in names
    for nm in names:
        assert hasattr(L, nm), nm
    assert sorted(P.EXPORTED_SYMBOLS) == names


def test_binding_methods_follow_the_header_names():
    for nm in declared_symbols():
        if nm in ("oci_create", "oci_destroy", "oci_last_error"):
            continue
        meth = nm if nm in ("oci_step", "si_step") else nm[len("oci_"):]
        assert hasattr(P.OCI, meth) or hasattr(P, meth), meth       # per-context calls are methods, the rest module functions


@pytest.mark.parametrize("N", [2, 4, 16, 64, 128, 256])
def test_device_library_quadrature_matches_numpy(N):
    g = P.OCI(np.ones(3), np.ones(3), np.full(3, 0.5), 1.0, 0.1, N)
    mu, w = g.get_quadrature()
    x, ww = np.polynomial.legendre.leggauss(N)
    assert np.max(np.abs(mu - x)) < 4e-16
    assert np.max(np.abs(w - ww)) < 2e-14
    assert abs(w.sum() - 2.0) < 1e-14 and np.all(np.diff(mu) > 0)
    g.close()


@pytest.mark.parametrize("kw", [
    dict(dx=[0.0, 1.0]), dict(dx=[-1.0, 1.0]), dict(st=[-0.1, 1.0]), dict(ss=[1.0, -2.0]), dict(v=0.0), dict(dt=0.0),
    dict(dt=float("nan")), dict(N=3), dict(N=0), dict(N=1), dict(N=514), dict(bcL=(7, 0.0)), dict(bcR=(1, float("inf"))),
    dict(dx=[float("nan"), 1.0]),
])
def test_create_rejects_invalid_arguments(kw):
    dx, st, ss = kw.get("dx", [1.0, 1.0]), kw.get("st", [1.0, 1.0]), kw.get("ss", [0.5, 0.5])
    with pytest.raises(P.OCIError) as e:
        P.OCI(dx, st, ss, kw.get("v", 1.0), kw.get("dt", 0.1), kw.get("N", 4), kw.get("bcL", (0, 0.0)), kw.get("bcR", (0, 0.0)))
    assert e.value.code == -1


def test_create_null_and_empty():
    L = P.load_library()
    h = C.c_void_p()
    one = (C.c_double * 1)(1.0)
    bc = P.binding._bc(0, 0.0)
    assert L.oci_create(None, 1, one, one, one, 1.0, 1.0, 2, bc, bc) == -1
    assert L.oci_create(C.byref(h), 0, one, one, one, 1.0, 1.0, 2, bc, bc) == -1
    assert L.oci_create(C.byref(h), 1, None, one, one, 1.0, 1.0, 2, bc, bc) == -1
    assert not h.value
    assert L.oci_workspace_bytes(None) == 0
    assert L.oci_launch_count(None) == 0
    assert L.oci_last_error(None) == b"NULL context"
    L.oci_destroy(None)


def test_classification_and_workspace_size():
    J, N = 50, 8
    n = 4 * N
    g = P.OCI(np.full(J, 0.1), np.ones(J), np.full(J, 0.9), 1.0, 0.1, N)
    i = g.get_info()
    assert (i["cells"], i["n_angles"], i["block_dim"], i["n_blocks"], i["path"]) == (J, N, n, 1, P.PATH_SHARED)
    ws = g.workspace_bytes()
    assert ws >= (n * n + 2 * (J + 2) * n + J * n) * 8 and ws % 256 == 0
    g.close()
    # bitwise-equal triples share a block; numbering by first appearance
    dx = np.array([0.1, 0.2, 0.1, 0.2, 0.3])
    h = P.OCI(dx, np.ones(5), np.full(5, 0.5), 1.0, 0.1, N)
    i = h.get_info()
    assert i["n_blocks"] == 3 and i["path"] == P.PATH_PER_CELL
    assert h.workspace_bytes() >= 3 * n * n * 8
    h.close()


def test_call_order_errors_without_device():
    L = P.load_library()
    g = P.OCI(np.ones(4), np.ones(4), np.full(4, 0.5), 1.0, 0.1, 4)
    it, res = C.c_int32(0), C.c_double(0.0)
    assert L.oci_step(g._h, 1e-10, 10, C.byref(it), C.byref(res)) == -2
    assert L.si_step(g._h, 1e-10, 10, C.byref(it), C.byref(res)) == -2
    assert b"oci_setup" in L.oci_last_error(g._h)
    buf = np.zeros(4 * 4 * 4)
    assert L.oci_set_flux(g._h, P.binding._hp(buf)) == -2
    assert L.oci_set_source(g._h, P.binding._hp(buf)) == -2
    assert L.oci_get_scalar_flux(g._h, P.binding._hp(buf)) == -2
    assert L.oci_get_block_inverse(g._h, 0, P.binding._hp(buf)) == -2
    assert L.oci_setup(g._h, None, 0, None) == -1
    assert L.oci_setup(g._h, C.c_void_p(128), 1 << 30, None) == -1       # not 256-byte aligned
    assert L.oci_setup(g._h, C.c_void_p(256), 16, None) == -5            # too small (never dereferenced)
    g.close()


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    g = P.OCI(np.ones(4), np.ones(4), np.full(4, 0.5), 1.0, 0.1, 4)
    with pytest.raises(P.OCIError) as e:
        g.setup()
    assert e.value.code == -3
    g.close()


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2305_13555_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.lower() or f == "__init__.py" and "import" not in txt.lower().split("oracle")[0][-40:], (dirpath, f)
