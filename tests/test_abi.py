"""The C-ABI library loads on a machine without a GPU and exports every symbol include/jxs.h
declares; without a device the product path fails loudly (no CPU fallback).  -m "not gpu"."""
import ctypes as C
import os
import re

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    src = open(os.path.join(ROOT, "include", "jxs.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(jxs_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_the_calls_of_the_north_star():
    names = declared_functions()
    for n in ("jxs_create", "jxs_set_ibm", "jxs_rhs", "jxs_max_wavespeed", "jxs_step", "jxs_set_flux_mlp"):
        assert n in names


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_2601_04400_b200 import jxs
    L = jxs.lib()
    names = declared_functions()
    assert len(names) >= 15
    for n in names:
        assert hasattr(L, n), n
    assert sorted(jxs.EXPORTS) == names  # the binding names every call of the header


def test_binding_does_not_import_the_oracle():
    import subprocess
    import sys
    code = ("import sys; import paper_2601_04400_b200.jxs, paper_2601_04400_b200.workloads; "
            "assert not any(m == 'oracle' or m.startswith('oracle.') for m in sys.modules), 'oracle imported'")
    subprocess.run([sys.executable, "-c", code], check=True, cwd=ROOT)


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU failure mode")
def test_no_device_fails_loudly():
    from paper_2601_04400_b200 import jxs
    bc = dict(xlo="periodic", xhi="periodic", ylo="periodic", yhi="periodic")
    with pytest.raises(jxs.JxsError) as e:
        jxs.Solver(16, 16, 0.1, 0.1, bc=bc)
    assert e.value.code == jxs.ECUDA
    # and straight through the C ABI
    h = C.c_void_p()
    b = jxs.make_bc(bc)
    rc = jxs.lib().jxs_create(16, 16, 0.1, 0.1, 1.4, 0.0, 0.72, C.byref(b), 0, None, C.byref(h))
    assert rc == jxs.ECUDA and not h.value


def test_argument_checks_do_not_need_a_device():
    from paper_2601_04400_b200 import jxs
    L = jxs.lib()
    h = C.c_void_p()
    b = jxs.make_bc(dict(xlo="periodic", xhi="transmissive", ylo="periodic", yhi="periodic"))
    assert L.jxs_create(16, 16, 0.1, 0.1, 1.4, 0.0, 0.72, C.byref(b), 0, None, C.byref(h)) == jxs.EINVAL
    b = jxs.make_bc(dict(xlo="periodic", xhi="periodic", ylo="periodic", yhi="periodic"))
    assert L.jxs_create(4, 16, 0.1, 0.1, 1.4, 0.0, 0.72, C.byref(b), 0, None, C.byref(h)) == jxs.EINVAL
    assert L.jxs_create(16, 16, -0.1, 0.1, 1.4, 0.0, 0.72, C.byref(b), 0, None, C.byref(h)) == jxs.EINVAL
    assert L.jxs_create(16, 16, 0.1, 0.1, 1.0, 0.0, 0.72, C.byref(b), 0, None, C.byref(h)) == jxs.EINVAL
    assert L.jxs_create(16, 16, 0.1, 0.1, 1.4, 1e-3, 0.0, C.byref(b), 0, None, C.byref(h)) == jxs.EINVAL
    assert L.jxs_create(16, 16, 0.1, 0.1, 1.4, 0.0, 0.72, C.byref(b), 7, None, C.byref(h)) == jxs.EINVAL
    assert L.jxs_create(16, 16, 0.1, 0.1, 1.4, 0.0, 0.72, None, 0, None, C.byref(h)) == jxs.EINVAL
    assert L.jxs_step(None, None, 0.4, 1) == jxs.EINVAL
    assert L.jxs_last_error(None) == b"null handle"


def test_argument_checks_of_the_next_rows():
    """one-dimensional path and the entry points added for SURVEY.md section 8(f): checks that need no device"""
    from paper_2601_04400_b200 import jxs
    L = jxs.lib()
    h = C.c_void_p()
    b = jxs.make_bc(dict(xlo="transmissive", xhi="transmissive", ylo="transmissive", yhi="transmissive"))
    assert L.jxs_create(64, 5, 0.1, 0.1, 1.4, 0.0, 0.72, C.byref(b), 0, None, C.byref(h)) == jxs.EINVAL   # 1 < ny < 8
    assert L.jxs_create(64, 1, 0.1, 0.1, 1.4, 1e-3, 0.0, C.byref(b), 0, None, C.byref(h)) == jxs.EINVAL   # Pr with mu > 0
    assert L.jxs_create(4, 1, 0.1, 0.1, 1.4, 0.0, 0.72, C.byref(b), 0, None, C.byref(h)) == jxs.EINVAL
    assert L.jxs_step_async(None, None, 0.4, 1) == jxs.EINVAL
    assert L.jxs_wait(None) == jxs.EINVAL
    assert L.jxs_set_time_integrator(None, 0) == jxs.EINVAL


def test_one_dimensional_workload_is_the_planar_one():
    import numpy as np
    from paper_2601_04400_b200 import workloads as wl
    c1, c2 = wl.sod1d(128), wl.sod(128, 128, 0)
    assert c1["U0"].shape == (4, 1, 128) and c1["ny"] == 1 and c1["dy"] == c1["dx"]
    assert np.array_equal(c1["U0"][:, 0], c2["U0"][:, 17])
    rows = wl.as_rows(c1)
    assert rows["U0"].shape == (4, 8, 128) and rows["bc"]["ylo"] == "periodic" and rows["bc"]["xlo"] == "transmissive"
    assert all(np.array_equal(rows["U0"][:, j], c1["U0"][:, 0]) for j in range(8))
