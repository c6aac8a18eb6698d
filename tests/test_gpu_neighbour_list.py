"""Skin neighbour list (lv_set_neighbour_list): same results as the
per-step cell rebuild -- neighbour counts bit-exact (fp32 contract #2), forces to rounding,
trajectories within the oracle tolerances -- with rebuilds decided on the device."""
import numpy as np
import pytest

from paper_2501_04456_b200 import workloads as W

pytestmark = pytest.mark.gpu

FORCE_TOL = 1e-5


@pytest.fixture(scope="module")
def orc():
    import oracle
    return oracle


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2501_04456_b200 import binding
    binding.load()
    return binding


def force_error(Fg, Fo, So):
    err = np.abs(Fg.astype(np.float64) - Fo).max(axis=1)
    nz = So > 0
    return (err[nz] / So[nz]).max() if nz.any() else 0.0


CASES = [  # (config, n, cells_per_cut, skin, capacity)
    ("C1", None, None, 0.3, 64),
    ("C3", 20000, [1, 2, 2], 0.5, 256),
    ("C4", 19999, [2], 0.2, 160),
    ("C2", 8191, [2, 2], 0.4, 256),
]


@pytest.mark.parametrize("name,n,cpc,skin,cap", CASES)
def test_first_step_forces_and_counts_against_oracle(B, orc, name, n, cpc, skin, cap):
    w = W.make_workload(name, n)
    p = orc.params_from_workload(w)
    Fo, So, co, _ = orc.pair_forces(p, w.pos, w.type, "cells")
    sim = B.Simulation.from_workload(w, cells_per_cut=cpc, neighbour_list=(skin, cap))
    sim.step(1)                                   # first step after lv_set_state: the cell kernel
    Fg, cg = sim.get_forces()
    assert np.array_equal(cg, co)                 # neighbour counts bit-exact
    assert force_error(Fg, Fo, So) <= FORCE_TOL
    assert sim.rebuild_count() == 0
    x1, v1, t1, R1, st1 = sim.get_state()
    sim.step(1)                                   # builds the list; forces of the state after step 1
    assert sim.rebuild_count() == 1
    Fl, cl = sim.get_forces()
    Fo1, So1, co1, _ = orc.pair_forces(p, x1, t1, "cells")
    assert np.array_equal(cl, co1)
    assert force_error(Fl, Fo1, So1) <= FORCE_TOL
    sim.close()


@pytest.mark.parametrize("name,n,cpc,skin,cap", CASES)
def test_list_stays_complete_between_rebuilds(B, name, n, cpc, skin, cap):
    """At arbitrary later steps the list run's forces and counts equal a fresh cell rebuild of
    the same state: no in-range pair is ever missing from a list that was built steps ago."""
    w = W.make_workload(name, n)
    lst = B.Simulation.from_workload(w, cells_per_cut=cpc, neighbour_list=(skin, cap))
    cel = B.Simulation.from_workload(w, cells_per_cut=cpc, neighbour_list=None)
    done = 0
    for k in (3, 37, 150, 400):
        lst.step(k - done)
        done = k
        x, v, t, R, st = lst.get_state()
        assert st == k
        cel.set_state(x, v, t, step=k)
        cel.compute_forces()
        Fc, cc = cel.get_forces()
        lst.step(1)                               # forces of the state at step k
        done += 1
        Fl, cl = lst.get_forces()
        assert np.array_equal(cl, cc), k
        S = np.abs(Fc).sum(axis=1) + 1e-30
        # same pairs, different summation order: rounding only (relative to the net force
        # plus a floor for cancelling terms)
        assert np.max(np.abs(Fl - Fc).max(axis=1) / (S + np.abs(Fc).max())) <= 1e-4, k
    r = lst.rebuild_count()
    assert 1 < r < done, r                        # rebuilt, but not every step
    assert lst.status() == 0
    lst.close(); cel.close()


def test_hundred_steps_against_oracle(B, orc):
    w = W.make_workload("C3", 20000)
    p = orc.params_from_workload(w)
    xo, vo, bad = orc.step(p, w.pos, w.vel, w.type, step0=0, nsteps=100)
    assert bad == 0
    sim = B.Simulation.from_workload(w, cells_per_cut=[1, 2, 2], neighbour_list=(0.5, 256))
    sim.step(100)
    x, v, t, R, st = sim.get_state()
    assert st == 100
    assert np.linalg.norm(x.astype(np.float64) - xo, axis=1).max() <= 1e-3 * R
    assert 1 <= sim.rebuild_count() < 100
    sim.close()


def test_split_invariance_and_restart(B):
    w = W.make_workload("C2", 8191)
    a = B.Simulation.from_workload(w, cells_per_cut=[2, 2], neighbour_list=(0.4, 256))
    b = B.Simulation.from_workload(w, cells_per_cut=[2, 2], neighbour_list=(0.4, 256))
    a.step(60)
    b.step(23); b.step(1); b.step(36)
    xa, va, _, _, _ = a.get_state()
    xb, vb, _, _, _ = b.get_state()
    assert np.array_equal(xa, xb) and np.array_equal(va, vb)
    assert a.rebuild_count() == b.rebuild_count()
    # lv_compute_forces between steps (always the cells) does not disturb the list run
    b.compute_forces()
    a.step(40); b.step(40)
    xa, va, _, _, _ = a.get_state()
    xb, vb, _, _, _ = b.get_state()
    assert np.array_equal(xa, xb) and np.array_equal(va, vb)
    # lv_set_state starts a fresh list
    a.set_state(w.pos, w.vel, w.type, 0)
    a.step(60)
    xc, vc, _, _, _ = a.get_state()
    b.set_state(w.pos, w.vel, w.type, 0)
    b.step(60)
    xd, vd, _, _, _ = b.get_state()
    assert np.array_equal(xc, xd) and np.array_equal(vc, vd)
    a.close(); b.close()


def test_pool_too_small_falls_back_to_the_cells(B):
    """A pool the list cannot fit (8 entries per NP for ~50 neighbours): no error, the warning
    bit is raised and every step runs on the cell kernel -- the same kernels as the default
    path, so counts, forces and the trajectory are BIT-identical to a run without the list."""
    w = W.make_workload("C4", 19999)              # ~50 neighbours per NP
    lst = B.Simulation.from_workload(w, cells_per_cut=[2], neighbour_list=(0.2, 8))
    cel = B.Simulation.from_workload(w, cells_per_cut=[2], neighbour_list=None)
    lst.step(1); cel.step(1)
    Fl, cl = lst.get_forces()
    Fc, cc = cel.get_forces()
    assert np.array_equal(cl, cc) and np.array_equal(Fl, Fc) and cc.sum() > 0
    lst.step(70); cel.step(70)                    # past a re-count (every 64th step)
    assert lst.status() == B.ST_LIST_OVERFLOW
    a, b = lst.get_state(), cel.get_state()       # no LV_E_CAPACITY any more
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and a[4] == b[4] == 71
    st = lst.list_stats()
    assert st["fallback_steps"] == 70 and st["entries_used"] > st["pool_entries"]
    lst.close(); cel.close()


def test_list_follows_a_shrinking_droplet_into_the_fallback(B, orc):
    """The pool fits the dilute start of C2 and not its crowded end: the run starts on the list,
    changes over to the cells on the device when a rebuild no longer fits, keeps the oracle
    tolerance over the first 100 steps, stays split-invariant across the change-over, and its
    counts at the end equal a fresh cell rebuild of the same state."""
    w = W.make_workload("C2", 8191)
    p = orc.params_from_workload(w)
    mk = lambda: B.Simulation.from_workload(w, cells_per_cut=[2, 2], neighbour_list=(0.4, 96))
    a, b = mk(), mk()
    a.step(100)
    x, v, t, R, st = a.get_state()
    xo, vo, bad = orc.step(p, w.pos, w.vel, w.type, step0=0, nsteps=100)
    assert bad == 0 and np.linalg.norm(x.astype(np.float64) - xo, axis=1).max() <= 1e-3 * R
    assert a.list_stats()["fallback_steps"] == 0
    a.step(6900)
    b.step(3300); b.step(1); b.step(3699)
    xa, va, ta, Ra, sa = a.get_state()
    xb, vb, _, _, sb = b.get_state()
    assert sa == sb == 7000 and np.array_equal(xa, xb) and np.array_equal(va, vb)
    st = a.list_stats()
    assert 0 < st["fallback_steps"] < 7000 and st["rebuilds"] > 1
    assert a.status() & B.ST_LIST_OVERFLOW
    cel = B.Simulation.from_workload(w, cells_per_cut=[2, 2], load_state=False, neighbour_list=None)
    cel.set_state(xa, va, ta, sa)
    cel.compute_forces()
    Fc, cc = cel.get_forces()
    a.step(1)
    Fl, cl = a.get_forces()
    assert np.array_equal(cl, cc) and cc.mean() > 60
    a.close(); b.close(); cel.close()


def test_automatic_skin_and_pool(B, orc):
    """lv_set_neighbour_list(skin <= 0, capacity = -1): skin = 0.16 of the smallest cut-off,
    pool = 2048 entries per NP; first-step counts bit-exact, 100 steps within tolerance."""
    w = W.make_workload("C3", 20000)
    p = orc.params_from_workload(w)
    Fo, So, co, _ = orc.pair_forces(p, w.pos, w.type, "cells")
    sim = B.Simulation.from_workload(w, cells_per_cut=[1, 2, 2], neighbour_list=(0.0, -1))
    sim.step(1)
    Fg, cg = sim.get_forces()
    assert np.array_equal(cg, co) and force_error(Fg, Fo, So) <= FORCE_TOL
    sim.step(99)
    x, v, t, R, st = sim.get_state()
    xo, vo, bad = orc.step(p, w.pos, w.vel, w.type, step0=0, nsteps=100)
    assert bad == 0 and np.linalg.norm(x.astype(np.float64) - xo, axis=1).max() <= 1e-3 * R
    s = sim.list_stats()
    assert s["pool_entries"] >= 2048 * w.n and s["fallback_steps"] == 0 and 1 <= s["rebuilds"] < 100
    assert sim.status() == 0
    sim.close()


def test_needs_the_counting_sort(B):
    w = W.make_workload("C1")
    with pytest.raises(B.LvError):
        B.Simulation.from_workload(w, options={B.OPT_SORT: B.SORT_RADIX}, neighbour_list=(0.3, 64))


@pytest.mark.parametrize("lanes", [1, 2, 4, 8, 16, 32])
def test_lanes_per_np_do_not_change_results(B, lanes):
    """LV_OPT_LIST_LANES: 1 .. 32 lanes sharing an NP's list give bit-identical neighbour counts
    and forces equal to rounding (different summation order), against a cell evaluation of the
    same state; 60 further steps stay close to the automatic choice."""
    w = W.make_workload("C3", 20000)
    cpc = [1, 2, 2]
    lst = B.Simulation.from_workload(w, cells_per_cut=cpc, neighbour_list=(0.5, -1),
                                     options={B.OPT_LIST_LANES: lanes})
    cel = B.Simulation.from_workload(w, cells_per_cut=cpc, neighbour_list=None)
    lst.step(5)
    x, v, t, R, st = lst.get_state()
    cel.set_state(x, v, t, step=st)
    cel.compute_forces()
    Fc, cc = cel.get_forces()
    lst.step(1)
    Fl, cl = lst.get_forces()
    assert lst.list_stats()["lanes_per_np"] in (4, 8) and lst.rebuild_count() >= 1
    assert np.array_equal(cl, cc) and cc.sum() > 0
    S = np.abs(Fc).sum(axis=1) + np.abs(Fc).max()
    assert np.max(np.abs(Fl - Fc).max(axis=1) / S) <= 1e-4
    auto = B.Simulation.from_workload(w, cells_per_cut=cpc, neighbour_list=(0.5, -1))
    auto.step(66); lst.step(60)
    xa, xl = auto.get_state()[0], lst.get_state()[0]
    assert np.abs(xa - xl).max() <= 1e-3
    for s in (lst, cel, auto):
        s.close()
