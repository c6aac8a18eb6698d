"""Host-side checks of the C-ABI library that need no GPU: it loads, exports
every symbol include/lv.h declares, validates arguments and call order, and its
host helpers agree with closed forms.  No compute call is made."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    from paper_2501_04456_b200 import binding
    binding.load()
    return binding


def test_exports_every_declared_symbol(B):
    hdr = open(os.path.join(ROOT, "include", "lv.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(lv_[a-z_0-9]+)\s*\(", hdr))
    assert declared == set(B.SYMBOLS)
    L = B.load()
    for name in declared:
        assert getattr(L, name) is not None
    assert b"sm_100a" in L.lv_version()


def test_struct_layouts_match_header(B):
    assert C.sizeof(B.LvType) == 7 * 8
    assert C.sizeof(B.GridInfo) == 4 + 32 + 36 + 32 + 32 + 64 + 256


def test_langevin_coeffs_closed_form(B):
    a, b = B.langevin_coeffs(2.0, 1.5, 3.0, 0.002)
    assert a == pytest.approx(1 - 2.0 * 0.002, rel=1e-15)
    # stationary variance of v' = a v + b xi is b^2/(1-a^2) = kT/m
    assert b * b / (1 - a * a) == pytest.approx(1.5 / 3.0, rel=1e-13)
    with pytest.raises(B.LvError):
        B.langevin_coeffs(1.0, 1.0, -1.0, 0.01)


def test_argument_and_order_errors(B):
    L = B.load()
    h = C.c_void_p()
    assert L.lv_create(C.byref(h), -1, 1, 0, 0.01) == -1
    assert L.lv_create(C.byref(h), 10, 0, 0, 0.01) == -1
    assert L.lv_create(C.byref(h), 10, 9, 0, 0.01) == -1
    assert L.lv_create(C.byref(h), 10, 1, 0, 0.0) == -1
    s = B.Simulation(10, 2, 1, 0.01)
    assert s.workspace_bytes() == 0                      # types not set yet
    assert L.lv_step(s.h, 1) == -2                        # not bound: order error
    assert L.lv_compute_forces(s.h) == -2
    assert L.lv_bind(s.h, None, 0, None) == -2
    t = [dict(sigma=1.0, mass=1.0), dict(sigma=-1.0, mass=1.0)]
    with pytest.raises(B.LvError):
        s.set_types(t)
    t[1]["sigma"] = 1.5
    with pytest.raises(B.LvError):                        # asymmetric table
        s.set_types(t, eps=[[1.0, 2.0], [3.0, 1.0]])
    s.set_types(t, eps=[[1.0, 2.0], [2.0, 1.0]], cut_factor=2.5)
    with pytest.raises(B.LvError):
        s.set_droplet_schedule(B.SCHED_LINEAR, 10.0, 5.0, 0)
    with pytest.raises(B.LvError):
        s.set_forces(0.0, (0, 0, 0), 7)
    with pytest.raises(B.LvError):
        s.set_grid([0, 1])
    s.set_droplet_schedule(B.SCHED_LINEAR, 10.0, 5.0, 100)
    assert s.workspace_bytes() > 10 * 96
    assert L.lv_bind(s.h, None, 1 << 30, None) == -3      # null / misaligned workspace
    assert L.lv_strerror(-3) == b"workspace too small or misaligned"
    assert L.lv_strerror(-5) == b"non-finite position or velocity"
    s.close()


def test_grid_info_follows_design_rule(B):
    """lv_get_debug(GRID) is host-only, so the grid rule can be checked here:
    h_b = r_c,bb (1+2^-9)/k_b; cover 2 R_max + 2 sigma_max; w_ab reaches r_c,ab."""
    s = B.Simulation(10, 2, 1, 0.01)
    s.set_types([dict(sigma=1.0, mass=1.0), dict(sigma=1.5, mass=3.0)], cut_factor=5.0)
    s.set_droplet_schedule(B.SCHED_LINEAR, 60.0, 25.0, 100)
    s.set_grid([1, 2])
    assert s.workspace_bytes() > 0
    g = s.grid()
    rc = {(0, 0): 5.0, (0, 1): 6.25, (1, 0): 6.25, (1, 1): 7.5}
    for b, k in ((0, 1), (1, 2)):
        assert g.h[b] == pytest.approx(rc[(b, b)] * (1 + 2.0 ** -9) / k, rel=1e-15)
        assert g.G[b] * g.h[b] >= 123.0 > (g.G[b] - 1) * g.h[b]
        assert g.lo[b] == np.float32(-0.5 * g.G[b] * g.h[b])
        for a in (0, 1):
            w = g.w[a * 8 + b]
            assert w * g.h[b] >= rc[(a, b)] * (1 + 2.0 ** -10) > (w - 1) * g.h[b]
    assert g.base[1] == g.G[0] ** 3 and g.base[2] == g.G[0] ** 3 + g.G[1] ** 3
    s.close()


def test_no_cpu_fallback(B):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    s = B.Simulation(10, 1, 1, 0.01)
    s.set_types([dict(sigma=1.0, mass=1.0)])
    s.set_droplet_schedule(B.SCHED_CONST, 10.0)
    with pytest.raises(RuntimeError):
        s.bind()
    s.close()


def test_product_does_not_import_oracle():
    """The product path may not route through the oracle (or the reference)."""
    pkg = os.path.join(ROOT, "paper_2501_04456_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), f
                assert "lv_oracle" not in src and "/root/reference" not in src, f
