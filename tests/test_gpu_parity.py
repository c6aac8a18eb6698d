"""Parity of the CUDA path (through the C ABI, include/lv.h) with the fp64 CPU
oracle on the same seeded inputs.  Bars (BASELINE.json north_star; DESIGN.md
"Parity protocol"): cell keys, sort permutation, cell offsets and neighbour
counts BIT-EXACT; forces max_i |dF_i|_inf / S_i <= 1e-5; one-step velocities
and positions <= 1e-5 (relative to |v| + sqrt(kT/m), resp. R); 100 steps
<= 1e-3 R.  All tests need a GPU."""
import numpy as np
import pytest

from paper_2501_04456_b200 import tuning, workloads as W

pytestmark = pytest.mark.gpu

FORCE_TOL = 1e-5


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2501_04456_b200 import binding
    binding.load()
    return binding


CASES = [          # (config, n or None for full size, cells_per_cut)
    ("C1", None, None),
    ("C1", None, [2]),
    ("C2", 8192, None),
    ("C2", 8191, [2, 3]),
    ("C3", 20000, None),
    ("C3", 20000, [1, 2, 2]),
    ("C4", 20000, None),
    ("C4", 19999, [2]),
    ("C5", 20001, None),
    ("T8", None, None),                     # LV_MAX_TYPES coexisting types
    ("T8", 5003, [1, 2, 1, 2, 1, 2, 1, 3]),
]

_cache = {}


def workload(name, n):
    key = (name, n)
    if key not in _cache:
        _cache[key] = W.make_workload(name, n)
    return _cache[key]


def force_error(Fg, Fo, So):
    err = np.abs(Fg.astype(np.float64) - Fo).max(axis=1)
    zero = So == 0
    assert np.all(Fg[zero] == 0.0)
    return (err[~zero] / So[~zero]).max() if (~zero).any() else 0.0


@pytest.mark.parametrize("name,n,cpc", CASES)
def test_cell_structures_bit_exact(B, orc, name, n, cpc):
    w = workload(name, n)
    p = orc.params_from_workload(w)
    g = orc.grid_spec(p, cpc)
    sim = B.Simulation.from_workload(w, cells_per_cut=cpc)
    sim.compute_forces()
    gg = sim.grid()
    T = w.n_types
    assert gg.n_types == g.n_types
    for b in range(T):
        assert gg.G[b] == g.G[b] and gg.base[b] == g.base[b]
        assert np.float32(gg.lo[b]).tobytes() == np.float32(g.lo[b]).tobytes()
        assert np.float32(gg.inv_h[b]).tobytes() == np.float32(g.inv_h[b]).tobytes()
        assert gg.h[b] == g.h[b]
        for a in range(T):
            assert gg.w[a * 8 + b] == g.w[a * 8 + b]
    assert gg.base[T] == g.base[T]
    key, ks, perm, off = orc.cell_structures(g, w.pos, w.type)
    assert np.array_equal(sim.get_debug(B.DBG_KEYS), key)
    assert np.array_equal(sim.get_debug(B.DBG_KEYS_SORTED), ks)
    assert np.array_equal(sim.get_debug(B.DBG_PERM), perm)
    assert np.array_equal(sim.get_debug(B.DBG_CELL_OFFSETS), off)
    assert np.array_equal(sim.get_debug(B.DBG_IDS_SORTED), perm)   # slot = id after set_state
    assert sim.status() == 0
    sim.close()


@pytest.mark.parametrize("name,n,cpc", CASES)
def test_forces_and_counts(B, orc, name, n, cpc):
    w = workload(name, n)
    p = orc.params_from_workload(w)
    Fo, So, co, _ = orc.pair_forces(p, w.pos, w.type, "cells")
    sim = B.Simulation.from_workload(w, cells_per_cut=cpc)
    sim.compute_forces()
    Fg, cg = sim.get_forces()
    assert np.array_equal(cg, co)                     # neighbour counts bit-exact
    assert co.sum() > 0
    assert force_error(Fg, Fo, So) <= FORCE_TOL
    # Newton III on the GPU result itself
    assert np.all(np.abs(Fg.astype(np.float64).sum(axis=0)) <= 1e-5 * So.sum())
    sim.close()


@pytest.mark.parametrize("name", ["C3", "C4", "C5"])
def test_forces_full_size(B, orc, name):
    """BASELINE sizes (N = 2.5e5, 2^20) in the launch configuration bench.py times
    (default force kernel, the workload's tuned cells_per_cut)."""
    w = workload(name, None)
    p = orc.params_from_workload(w)
    Fo, So, co, _ = orc.pair_forces(p, w.pos, w.type, "cells")
    sim = B.Simulation.from_workload(w, cells_per_cut=tuning.cells_per_cut(w))
    sim.compute_forces()
    Fg, cg = sim.get_forces()
    assert np.array_equal(cg, co)
    assert force_error(Fg, Fo, So) <= FORCE_TOL
    ks = sim.get_debug(B.DBG_KEYS_SORTED)
    assert np.all(np.diff(ks.astype(np.int64)) >= 0)
    assert np.array_equal(np.sort(sim.get_debug(B.DBG_PERM)), np.arange(w.n, dtype=np.uint32))
    off = sim.get_debug(B.DBG_CELL_OFFSETS)
    assert off[0] == 0 and off[-1] == w.n and np.all(np.diff(off.astype(np.int64)) >= 0)
    sim.close()


def test_dense_compressed_state(B, orc):
    """A crowded state (C2 pushed to its final radius): hundreds of NPs per
    cell, long rows."""
    w = W.make_workload("C2", 8192)
    f = 0.55
    w.pos = (w.pos * np.float32(f)).astype(np.float32)
    w.R0 *= f
    w.R1 *= f
    p = orc.params_from_workload(w)
    Fo, So, co, _ = orc.pair_forces(p, w.pos, w.type, "cells")
    sim = B.Simulation.from_workload(w)
    sim.compute_forces()
    Fg, cg = sim.get_forces()
    assert np.array_equal(cg, co) and co.mean() > 150
    assert force_error(Fg, Fo, So) <= FORCE_TOL
    sim.close()


def vel_pos_check(w, p_orc, xo, vo, xg, vg, S_pair, R):
    m = np.asarray(w.mass)[w.type]
    vscale = np.linalg.norm(vo, axis=1) + np.sqrt(w.kT / m)
    dv = np.abs(vg.astype(np.float64) - vo).max(axis=1)
    tol_v = 1e-5 * vscale + (w.dt / m) * FORCE_TOL * S_pair
    assert np.all(dv <= tol_v), float((dv / tol_v).max())
    dx = np.abs(xg.astype(np.float64) - xo).max(axis=1)
    assert dx.max() / R <= 1e-5


@pytest.mark.parametrize("name,n", [("C1", None), ("C2", 8192), ("C3", 20000), ("C4", 20000), ("C5", 20001),
                                    ("T8", None)])
def test_one_step(B, orc, name, n):
    w = workload(name, n)
    p = orc.params_from_workload(w)
    xo, vo, bad = orc.step(p, w.pos, w.vel, w.type, step0=0, nsteps=1)
    _, So, _, _ = orc.pair_forces(p, w.pos, w.type, "cells")
    sim = B.Simulation.from_workload(w)
    sim.step(1)
    xg, vg, tg, R, st = sim.get_state()
    assert bad == 0 and st == 1
    assert np.array_equal(tg, w.type)
    assert R == pytest.approx(orc.radius(p, 1), rel=1e-15)
    vel_pos_check(w, p, xo, vo, xg, vg, So, R)
    sim.close()


def test_one_step_moving_interface_near_wall(B, orc):
    """A step taken after the interface has moved 0.8 sigma into the initial
    distribution: hundreds of NPs are pressed by the surface spring, the
    surface term dominates and |x| - (R - r) is a cancellation (fp64
    sub-expression on the GPU).  Positions are untouched, so no pair overlaps."""
    w = W.make_workload("C3", 20000)
    step0 = int(0.8 / (w.R0 - w.R1) * w.sched_steps)
    p = orc.params_from_workload(w)
    xo, vo, bad, Fp, Fe = orc.step(p, w.pos, w.vel, w.type, step0=step0, nsteps=1, want_forces=True)
    assert bad == 0
    assert (np.abs(Fe).max(axis=1) > 1.0).sum() > 500        # the wall is really felt
    _, So, _, _ = orc.pair_forces(p, w.pos, w.type, "cells")
    Sw = np.abs(Fe).sum(axis=1)
    sim = B.Simulation.from_workload(w, load_state=False)
    sim.set_state(w.pos, w.vel, w.type, step0)
    sim.step(1)
    xg, vg, _, Rg, st = sim.get_state()
    assert st == step0 + 1 and Rg == pytest.approx(orc.radius(p, step0 + 1), rel=1e-15)
    vel_pos_check(w, p, xo, vo, xg, vg, So + Sw, Rg)
    sim.close()


@pytest.mark.parametrize("name,n,cpc", [("C1", None, None), ("C2", 8192, None), ("C4", 8000, None),
                                        ("T8", 6000, None), ("C3", 20000, [1, 2, 2]), ("C5", 20001, None),
                                        ("C3", None, "tuned")])
def test_hundred_steps(B, orc, name, n, cpc):
    """100 steps on the DEFAULT path (north_star: "states after 100 steps within 1e-3 of the
    droplet radius"), C3 -- the bench workload -- also at full size with its tuned grids."""
    w = workload(name, n)
    if cpc == "tuned":
        cpc = tuning.cells_per_cut(w)
    p = orc.params_from_workload(w)
    xo, vo, bad = orc.step(p, w.pos, w.vel, w.type, step0=0, nsteps=100)
    sim = B.Simulation.from_workload(w, cells_per_cut=cpc)
    sim.step(100)
    xg, vg, _, R, st = sim.get_state()
    assert bad == 0 and st == 100
    assert R == pytest.approx(orc.radius(p, 100), rel=1e-15)
    d = np.linalg.norm(xg.astype(np.float64) - xo, axis=1)
    assert d.max() <= 1e-3 * R, d.max() / R
    assert sim.status() == 0
    sim.close()


def test_forces_at_the_benched_snapshots(B, orc):
    """The later states bench.py times (C3, N = 2.5e5, tuned grids, steps 10 000 and 17 000 of
    the shrinking schedule: ~210 and ~580 in-range neighbours per NP): the GPU's own state at
    those steps goes to both sides; neighbour counts bit-exact, forces to 1e-5 S, with the
    default kernel and with the shared-candidate-stream kernel."""
    w = workload("C3", None)
    p = orc.params_from_workload(w)
    cpc = tuning.cells_per_cut(w)
    sim = B.Simulation.from_workload(w, cells_per_cut=cpc)
    tile = B.Simulation.from_workload(w, cells_per_cut=cpc, load_state=False,
                                      options={B.OPT_FORCE_KERNEL: B.FORCE_TILE, B.OPT_TILE_SUBSTREAMS: 8})
    cur = 0
    for target, lo in ((10000, 150), (17000, 400)):
        sim.step(target - cur)
        cur = target
        x, v, t, R, st = sim.get_state()
        assert st == target and sim.status() == 0
        Fo, So, co, _ = orc.pair_forces(p, x, t, "cells")
        assert co.mean() > lo
        sim.compute_forces()
        Fg, cg = sim.get_forces()
        assert np.array_equal(cg, co)
        assert force_error(Fg, Fo, So) <= FORCE_TOL
        tile.set_state(x, v, t, st)
        tile.compute_forces()
        Ft, ct = tile.get_forces()
        assert np.array_equal(ct, co)
        assert force_error(Ft, Fo, So) <= FORCE_TOL
    sim.close(); tile.close()


@pytest.mark.parametrize("name,n,cpc", [("C2", 8192, [2, 2]), ("C3", 20000, [1, 2, 2]), ("C4", 8000, None)])
def test_steady_state_permutation_against_the_oracle(B, orc, name, n, cpc):
    """fp32 contract #3 in steady state (hash fused into the update kernel, CUDA-graph replay):
    the slot order of step k + 1 must be the STABLE sort, by the oracle's cell keys of the
    positions after step k, of the slot order of step k."""
    w = workload(name, n)
    p = orc.params_from_workload(w)
    g = orc.grid_spec(p, cpc)
    sim = B.Simulation.from_workload(w, cells_per_cut=cpc, neighbour_list=None)    # the cells, every step
    sim.step(5)
    ids_prev = sim.get_debug(B.DBG_IDS_SORTED).astype(np.int64)
    moved = 0
    for k in range(20):
        x, v, t, R, st = sim.get_state()              # state the next step starts from, by id
        key, ks, perm, off = orc.cell_structures(g, x[ids_prev], t[ids_prev])
        sim.step(1)
        ids_next = sim.get_debug(B.DBG_IDS_SORTED).astype(np.int64)
        assert np.array_equal(ids_next, ids_prev[perm.astype(np.int64)])
        moved += int((ids_next != ids_prev).sum())
        ids_prev = ids_next
    assert moved > 0                                   # NPs did change cells meanwhile
    sim.close()


def test_one_step_late_schedule_near_wall(B, orc):
    """Late in the schedule many NPs are pressed against the moving interface: the GPU runs
    C3@20000 to step 6 000, that state goes to both sides, one step to the one-step bars (the
    wall term in the force scale)."""
    w = workload("C3", 20000)
    p = orc.params_from_workload(w)
    run = B.Simulation.from_workload(w, cells_per_cut=[1, 2, 2])
    run.step(6000)
    x, v, t, R, st = run.get_state()
    assert st == 6000 and run.status() == 0
    run.close()
    xo, vo, bad, Fp, Fe = orc.step(p, x, v, t, step0=st, nsteps=1, want_forces=True)
    assert bad == 0
    assert (np.abs(Fe).max(axis=1) > 1.0).sum() > 300         # the wall is really felt
    _, So, _, _ = orc.pair_forces(p, x, t, "cells")
    Sw = np.abs(Fe).sum(axis=1)
    sim = B.Simulation.from_workload(w, load_state=False)
    sim.set_state(x, v, t, st)
    sim.step(1)
    xg, vg, _, Rg, st1 = sim.get_state()
    assert st1 == st + 1 and Rg == pytest.approx(orc.radius(p, st + 1), rel=1e-15)
    vel_pos_check(w, p, xo, vo, xg, vg, So + Sw, Rg)
    sim.close()


def test_forces_survive_an_observe_call(B):
    """lv_get_forces after lv_step + lv_observe_*: the observables re-sort the B copy, the
    forces of the last step must still be attributed to the right NPs."""
    w = workload("C2", 8192)
    sim = B.Simulation.from_workload(w)
    sim.step(25)
    F0, c0 = sim.get_forces()
    sim.observe_rdf(0.05, 100)
    F1, c1 = sim.get_forces()
    sim.observe_clusters(1.5)
    F2, c2 = sim.get_forces()
    assert np.array_equal(F0, F1) and np.array_equal(c0, c1)
    assert np.array_equal(F0, F2) and np.array_equal(c0, c2)
    assert c0.sum() > 0
    sim.close()


@pytest.mark.parametrize("fk,sub", [(0, None), (1, None), (2, None), (3, None), (4, 1), (4, 8)])
def test_bonded_pair_outside_the_grid(B, orc, fk, sub):
    """NPs beyond the grid are clamped into the border cells (R22, warning only): two bonded
    NPs outside along +x, two along -x and two along +y must still see each other, in every
    force kernel and through the neighbour list."""
    w = W.make_workload("C1", None)
    p = orc.params_from_workload(w)
    pos = w.pos.copy()
    far = 40.0                                   # grid half-width ~ 22.5
    pos[0] = [far, 0.3, 0.2];  pos[1] = [far + 1.1, 0.3, 0.2]
    pos[2] = [-far, -0.4, 0.1]; pos[3] = [-far - 1.05, -0.4, 0.1]
    pos[4] = [0.5, far, 0.0];  pos[5] = [0.5, far + 1.2, 0.0]
    Fo, So, co, _ = orc.pair_forces(p, pos, w.type, "brute")
    assert np.all(co[:6] == 1)
    opts = {B.OPT_FORCE_KERNEL: fk}
    if sub is not None:
        opts[B.OPT_TILE_SUBSTREAMS] = sub
    sim = B.Simulation.from_workload(w, load_state=False, options=opts)
    sim.set_state(pos, w.vel, w.type, 0)
    sim.compute_forces()
    Fg, cg = sim.get_forces()
    assert sim.status() == B.ST_OUTSIDE_GRID
    assert np.array_equal(cg, co)
    assert force_error(Fg, Fo, So) <= FORCE_TOL
    sim.close()
    if fk == 2:
        lst = B.Simulation.from_workload(w, load_state=False, neighbour_list=(0.3, 64))
        lst.set_state(pos, np.zeros_like(w.vel), w.type, 0)
        lst.step(1)
        Fl, cl = lst.get_forces()
        assert np.array_equal(cl, co)
        # ... and through the list itself (built at the second step): the moved state against
        # a fresh cell evaluation of it
        xs, vs, ts, _, s1 = lst.get_state()
        lst.step(1)
        Fl2, cl2 = lst.get_forces()
        cel = B.Simulation.from_workload(w, load_state=False)
        cel.set_state(xs, vs, ts, s1)
        cel.compute_forces()
        Fc2, cc2 = cel.get_forces()
        assert lst.rebuild_count() == 1 and np.array_equal(cl2, cc2) and cc2[:6].sum() >= 0
        cel.close()
        lst.close()


@pytest.mark.parametrize("mode", ["LINEAR", "R2LAW"])
def test_condensing_droplet(B, orc, mode):
    """The droplet may also grow ("evaporating or condensing"): R1 > R0.  The grid
    is sized for max(R0, R1); the wall recedes, so NPs pressed against it are released.  Cell
    structures bit-exact after the interface has moved, 100 steps within 1e-3 R."""
    from dataclasses import replace
    w0 = workload("C2", 8192)
    w = replace(w0, R1=1.3 * w0.R0, sched_steps=150,
                sched_mode=W.SCHED_LINEAR if mode == "LINEAR" else W.SCHED_R2LAW)
    p = orc.params_from_workload(w)
    assert orc.radius(p, 150) == pytest.approx(1.3 * w0.R0, rel=1e-15)
    assert orc.radius(p, 75) > w0.R0
    sim = B.Simulation.from_workload(w, cells_per_cut=[2, 2])
    sim.step(100)
    xg, vg, tg, R, st = sim.get_state()
    xo, vo, bad = orc.step(p, w.pos, w.vel, w.type, step0=0, nsteps=100)
    assert bad == 0 and st == 100
    assert R == pytest.approx(orc.radius(p, 100), rel=1e-15) and R > w0.R0
    d = np.linalg.norm(xg.astype(np.float64) - xo, axis=1)
    assert d.max() <= 1e-3 * R, d.max() / R
    # cell structures of the GPU's own state at step 100, on the grid of the larger radius
    sim.compute_forces()
    g = orc.grid_spec(p, [2, 2])
    key, ks, perm, off = orc.cell_structures(g, xg, tg)
    ks_g = sim.get_debug(B.DBG_KEYS_SORTED)
    assert np.array_equal(ks_g, ks)
    assert np.array_equal(sim.get_debug(B.DBG_CELL_OFFSETS), off)
    # after steps the slots are no longer in id order (ties keep SLOT order, contract #3), so
    # the permutation is compared through the cell of every NP id
    key_by_id = np.empty_like(key)
    key_by_id[sim.get_debug(B.DBG_IDS_SORTED)] = ks_g
    assert np.array_equal(key_by_id, key)
    Fg, cg = sim.get_forces()
    Fo, So, co, _ = orc.pair_forces(p, xg, tg, "cells")
    assert np.array_equal(cg, co)
    assert force_error(Fg, Fo, So) <= FORCE_TOL
    assert sim.status() == 0
    sim.close()


def test_full_size_trajectory_in_the_bench_configuration(B, orc):
    """C3 at N = 2.5e5 exactly as bench.py times it (default kernels, tuned cells_per_cut,
    CUDA-graph replay): one step to the one-step bars and 20 steps to 1e-3 R against the
    oracle, every NP compared by id."""
    w = workload("C3", None)
    p = orc.params_from_workload(w)
    sim = B.Simulation.from_workload(w, cells_per_cut=tuning.cells_per_cut(w))
    x1o, v1o, bad = orc.step(p, w.pos, w.vel, w.type, step0=0, nsteps=1)
    assert bad == 0
    sim.step(1)
    x, v, _, R, st = sim.get_state()
    assert st == 1
    assert np.abs(x.astype(np.float64) - x1o).max() <= 1e-5 * R
    xo, vo, bad = orc.step(p, x1o, v1o, w.type, step0=1, nsteps=19)
    assert bad == 0
    sim.step(19)
    x, v, _, R, st = sim.get_state()
    assert st == 20
    d = np.linalg.norm(x.astype(np.float64) - xo, axis=1)
    assert d.max() <= 1e-3 * R, d.max() / R
    m = np.asarray(w.mass)[w.type]
    assert np.abs(v.astype(np.float64) - vo).max() <= 1e-2 * np.sqrt(w.kT / m.min())
    sim.close()


@pytest.mark.parametrize("name", ["P1", "P8"])
def test_paper_shaped_scenarios(B, orc, name):
    """Table 1 shapes at full size: P1 = 10^4 NPs, range 4 sigma, isotropic
    centrifugal force, windowed wall; P8 = 39 500 + 1 500 NPs with a 6 : 1 size ratio, the
    non-Berthelot eps matrix and radius-square-law evaporation.  Cell structures and counts
    bit-exact, forces to 1e-5, 100 steps to 1e-3 R, with and without the neighbour list."""
    w = workload(name, None)
    p = orc.params_from_workload(w)
    cpc = tuning.cells_per_cut(w)
    g = orc.grid_spec(p, cpc)
    key, ks, perm, off = orc.cell_structures(g, w.pos, w.type)
    Fo, So, co, _ = orc.pair_forces(p, w.pos, w.type, "cells")
    sim = B.Simulation.from_workload(w, cells_per_cut=cpc)
    sim.compute_forces()
    assert np.array_equal(sim.get_debug(B.DBG_KEYS_SORTED), ks)
    assert np.array_equal(sim.get_debug(B.DBG_PERM), perm)
    assert np.array_equal(sim.get_debug(B.DBG_CELL_OFFSETS), off)
    Fg, cg = sim.get_forces()
    assert np.array_equal(cg, co) and co.sum() > 0
    assert force_error(Fg, Fo, So) <= FORCE_TOL
    xo, vo, bad = orc.step(p, w.pos, w.vel, w.type, step0=0, nsteps=100)
    assert bad == 0
    sim.step(100)
    x, v, _, R, st = sim.get_state()
    assert st == 100 and R == pytest.approx(orc.radius(p, 100), rel=1e-15)
    assert np.linalg.norm(x.astype(np.float64) - xo, axis=1).max() <= 1e-3 * R
    lst = B.Simulation.from_workload(w, cells_per_cut=cpc, neighbour_list=tuning.neighbour_list(w))
    lst.step(100)
    xl, vl, _, _, _ = lst.get_state()
    assert np.linalg.norm(xl.astype(np.float64) - xo, axis=1).max() <= 1e-3 * R
    assert 1 <= lst.rebuild_count() < 100
    sim.close(); lst.close()


def test_noise_matches_oracle_draws(B, orc):
    """a = 0, no forces, v0 = 0  ->  v1 = b xi: the GPU's Philox/Box-Muller
    draws against the oracle's, particle by particle, at a 64-bit step index."""
    n, b, seed, step0 = 5000, 0.75, 0xDEADBEEF12345678, (3 << 32) + 17
    sim = B.Simulation(n, 1, seed, 0.01)
    sim.set_types([dict(sigma=1.0, eps=0.0, mass=1.0, drag_a=0.0, kick_b=b)], cut_factor=40.0)
    sim.set_droplet_schedule(B.SCHED_CONST, 500.0)
    sim.bind()
    g = np.arange(18) * 50.0 - 425.0
    x0 = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)[:n].astype(np.float32)
    sim.set_state(x0, np.zeros((n, 3), np.float32), np.zeros(n, np.int32), step0)
    sim.step(1)
    _, v, _, _, st = sim.get_state()
    xi = orc.gauss3(seed, np.arange(n), step0)
    assert st == step0 + 1
    assert np.abs(v / b - xi).max() < 2e-6
    sim.close()


def test_split_invariance_and_roundtrip(B):
    w = workload("C2", 8192)
    s1 = B.Simulation.from_workload(w)
    s1.step(30)
    a = s1.get_state()
    s2 = B.Simulation.from_workload(w)
    s2.step(12)
    s2.step(18)
    b = s2.get_state()
    for u, v in zip(a[:3], b[:3]):
        assert np.array_equal(u, v)
    assert a[3:] == b[3:]
    # get -> set -> get is the identity (restart path)
    s3 = B.Simulation.from_workload(w, load_state=False)
    s3.set_state(a[0], a[1], a[2], a[4])
    c = s3.get_state()
    for u, v in zip(a[:3], c[:3]):
        assert np.array_equal(u, v)
    assert c[4] == 30
    # device-buffer variant of the accessors
    import torch
    pd, vd, td, R, st = s1.get_state(on_device=True)
    torch.cuda.synchronize()
    assert np.array_equal(pd.cpu().numpy(), a[0]) and np.array_equal(td.cpu().numpy(), a[2])
    s3.set_state(pd, vd, td, 30)
    c = s3.get_state()
    assert np.array_equal(c[0], a[0]) and np.array_equal(c[1], a[1])
    for s in (s1, s2, s3):
        s.close()


@pytest.mark.parametrize("batched", [True, False])
def test_replica_set_equals_solo_runs(B, orc, batched):
    """NEXT-3 batched replicas: R small droplets stepped together -- by ONE CUDA-graph launch
    per chunk of steps (lv_batch, parallel branches), or concurrently on R streams -- are each
    bit-identical to the same workload stepped alone (no coupling between replicas), differ from
    one another (distinct seeds), and replica 0 still tracks the oracle."""
    from paper_2501_04456_b200 import replicas
    mk = lambda seed: W.make_workload("C1", 1024, seed=seed)
    rs = replicas.ReplicaSet(mk, 5, base_seed=77, slice_steps=7, batched=batched, steps_per_launch=6)
    assert len(rs) == 5 and rs.n_particles == 5 * 1024
    rs.step(13)                      # two chunks of 6 and a single step
    rs.step(27)
    rs.synchronize()
    got = [rs.get_state(r) for r in range(5)]
    for r in range(5):
        solo = B.Simulation.from_workload(rs.workloads[r], cells_per_cut=tuning.cells_per_cut(rs.workloads[r]))
        solo.step(40)
        ref = solo.get_state()
        for u, v in zip(got[r][:3], ref[:3]):
            assert np.array_equal(u, v)
        assert got[r][3:] == ref[3:]
        solo.close()
    assert not np.array_equal(got[0][0], got[1][0])
    w0 = rs.workloads[0]
    p = orc.params_from_workload(w0)
    xo, vo, bad = orc.step(p, w0.pos, w0.vel, w0.type, step0=0, nsteps=40)
    assert bad == 0
    assert np.linalg.norm(got[0][0].astype(np.float64) - xo, axis=1).max() <= 1e-3 * got[0][3]
    rs.close()


def test_batched_replicas_with_neighbour_lists_equal_solo_runs(B):
    """lv_batch with the skin list on: every replica's steps sit in the one graph with their own
    IF node around the rebuild chain (replicas rebuild at different steps); each replica is
    bit-identical to the same workload stepped alone with the same list setting, and its list
    was rebuilt as often."""
    from paper_2501_04456_b200 import replicas
    mk = lambda seed: W.make_workload("C2", 3001, seed=seed)
    nl = (0.4, 256)
    rs = replicas.ReplicaSet(mk, 4, base_seed=5, batched=True, steps_per_launch=5, neighbour_list=nl)
    rs.step(3)
    rs.step(64)                      # chunks of 5 and single steps
    rs.synchronize()
    for r in range(4):
        got = rs.get_state(r)
        solo = B.Simulation.from_workload(rs.workloads[r], cells_per_cut=tuning.cells_per_cut(rs.workloads[r]),
                                          neighbour_list=nl)
        solo.step(67)
        ref = solo.get_state()
        for u, v in zip(got[:3], ref[:3]):
            assert np.array_equal(u, v)
        assert got[3:] == ref[3:]
        assert rs.sims[r].status() == 0
        ls, lr = rs.sims[r].list_stats(), solo.list_stats()
        assert ls["rebuilds"] == lr["rebuilds"] >= 2 and ls["fallback_steps"] == lr["fallback_steps"]
        solo.close()
    rs.close()


def test_restart_continues_within_tolerance(B):
    """Stop, save, restart: same noise (keyed on id and step);
    only the summation order changes, so the continuation agrees to rounding."""
    w = workload("C1", None)
    s1 = B.Simulation.from_workload(w)
    s1.step(20)
    mid = s1.get_state()
    s1.step(20)
    end = s1.get_state()
    s2 = B.Simulation.from_workload(w, load_state=False)
    s2.set_state(mid[0], mid[1], mid[2], mid[4])
    s2.step(20)
    end2 = s2.get_state()
    assert end2[4] == 40
    assert np.abs(end2[0] - end[0]).max() < 1e-4
    s1.close()
    s2.close()


@pytest.mark.parametrize("n", [0, 1, 2, 33, 129])
def test_tiny_and_empty(B, orc, n):
    rng = np.random.default_rng(n)
    x = (rng.uniform(-1.5, 1.5, size=(n, 3))).astype(np.float32)
    if n >= 2:
        g = np.arange(6) * 1.1 - 2.75
        x = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)[:n].astype(np.float32)
    v = rng.normal(0, 1, size=(n, 3)).astype(np.float32)
    t = np.zeros(n, np.int32)
    a, b = orc.langevin_coeffs(1.0, 1.0, 1.0, 0.005)
    p = orc.make_params(sigma=[1.0], mass=[1.0], charge=[0.0], wall_k=[100.0], drag_a=[a], kick_b=[b],
                        dt=0.005, eps=[1.0], cut_factor=2.5, R0=6.0, seed=5)
    sim = B.Simulation(n, 1, 5, 0.005)
    ga, gb = B.langevin_coeffs(1.0, 1.0, 1.0, 0.005)
    sim.set_types([dict(sigma=1.0, eps=1.0, mass=1.0, wall_k=100.0, drag_a=ga, kick_b=gb)], cut_factor=2.5)
    sim.set_droplet_schedule(B.SCHED_CONST, 6.0)
    sim.bind()
    sim.set_state(x, v, t, 0)
    sim.compute_forces()
    Fg, cg = sim.get_forces()
    Fo, So, co, _ = orc.pair_forces(p, x, t, "brute")
    assert np.array_equal(cg, co)
    if n:
        assert force_error(Fg, Fo, So) <= FORCE_TOL
    sim.step(3)
    xg, vg, tg, R, st = sim.get_state()
    xo, vo, _ = orc.step(p, x, v, t, nsteps=3, method="brute")
    assert st == (3 if n else 0) or n == 0
    if n:
        assert np.abs(xg - xo).max() < 1e-4 and np.abs(vg - vo).max() < 1e-3
    sim.close()


@pytest.mark.parametrize("n", [0, 1, 2])
def test_tiny_and_empty_observables_and_views(B, orc, n):
    """The rows built after the step (observables, aggregates, both views) on empty and tiny
    inputs: no crash, and the same answers as the oracle."""
    from oracle import observables as O
    x = np.array([[5.6, 0.0, 0.0], [4.5, 0.0, 0.0]], np.float32)[:n]     # one NP in the interface, a bonded pair
    t = np.zeros(n, np.int32)
    sim = B.Simulation(n, 1, 5, 0.005)
    ga, gb = B.langevin_coeffs(1.0, 1.0, 1.0, 0.005)
    sim.set_types([dict(sigma=1.0, eps=1.0, mass=1.0, wall_k=100.0, drag_a=ga, kick_b=gb)], cut_factor=2.5)
    sim.set_droplet_schedule(B.SCHED_CONST, 6.0)
    sim.bind()
    sim.set_state(x, np.zeros((n, 3), np.float32), t, 0)
    hist, g = sim.observe_rdf(0.1, 25)
    assert hist.sum() == (2 if n == 2 else 0)            # the ordered pair at r = 1.1, both ways
    assert np.array_equal(hist, orc.rdf_hist(x, 0.1, 25))
    rad = sim.observe_radial(0.5, 16)
    assert rad["hist"].sum() == n and rad["n_surf"] == (1 if n else 0)   # |x| = 5.6 > R - 2 r
    cl = sim.observe_clusters(1.5)
    assert cl["n_clusters"] == (1 if n else 0) and cl["largest"] == n
    if n:
        assert np.array_equal(cl["labels"], np.zeros(n, np.int32))
        assert np.array_equal(O.cluster_labels(x.astype(np.float64), t, [1.0]), np.zeros(n))
    pal = [0x00ff8040]
    img = sim.render(30.0, 200.0, 0.2, 0.1, 64, 48, pal, 0xff000000, 0xff201008)
    ref = orc.render(x, t, [0.5], 6.0, 30.0, 200.0, 0.2, 0.1, 64, 48, pal, 0xff000000, 0xff201008)
    assert np.array_equal(img, ref)
    smap = sim.render_surface(90, 45, pal, 0xff201008)
    sref = orc.render_surface(x, t, [0.5], 6.0, 90, 45, pal, 0xff201008)
    assert np.array_equal(smap, sref)
    assert ((smap != 0xff201008).sum() > 0) == (n >= 1)
    sim.close()


def test_status_flags(B):
    w = workload("C1", None)
    sim = B.Simulation.from_workload(w, load_state=False)
    pos = w.pos.copy()
    pos[7] = pos[8]                       # coincident pair: no core clamp (R6)
    sim.set_state(pos, w.vel, w.type, 0)
    sim.step(1)
    with pytest.raises(B.LvError) as e:
        sim.get_state()
    assert e.value.code == B.E_NONFINITE
    assert sim.status() & B.ST_NONFINITE
    # set_state clears the sticky bit
    sim.set_state(w.pos, w.vel, w.type, 0)
    sim.step(1)
    sim.get_state()
    assert sim.status() == 0
    # NaN injected
    pos = w.pos.copy()
    pos[100, 1] = np.nan
    sim.set_state(pos, w.vel, w.type, 0)
    sim.step(1)
    assert sim.status() & B.ST_NONFINITE
    # far outside the grid: warning only, forces still right for the others
    pos = w.pos.copy()
    pos[5] = [500.0, 0.0, 0.0]
    sim.set_state(pos, w.vel, w.type, 0)
    sim.compute_forces()
    assert sim.status() == B.ST_OUTSIDE_GRID
    sim.close()


def test_type_out_of_range_is_reported(B):
    """An NP type outside [0, n_types) would index the type tables out of range: it is loaded
    as type 0, LV_ST_BAD_TYPE is raised and lv_get_state returns LV_E_ARG."""
    w = workload("C2", 8192)
    sim = B.Simulation.from_workload(w, load_state=False)
    t = w.type.copy()
    t[17] = 2
    t[4000] = -1
    sim.set_state(w.pos, w.vel, t, 0)
    sim.step(2)
    assert sim.status() & 8
    with pytest.raises(B.LvError) as ei:
        sim.get_state()
    assert ei.value.code == -1
    sim.set_state(w.pos, w.vel, w.type, 0)      # a valid state clears the flag
    sim.step(2)
    assert sim.status() == 0
    sim.get_state()
    sim.close()


def test_wall_window_mode_and_r2law(B, orc):
    w = W.make_workload("C1", None)
    w.wall_mode = W.WALL_WINDOW
    w.sched_mode, w.R1, w.sched_steps = W.SCHED_R2LAW, 12.0, 50
    p = orc.params_from_workload(w)
    xo, vo, bad = orc.step(p, w.pos, w.vel, w.type, step0=0, nsteps=40)
    sim = B.Simulation.from_workload(w)
    sim.step(40)
    xg, vg, _, R, st = sim.get_state()
    assert R == pytest.approx(orc.radius(p, 40), rel=1e-14)
    d = np.linalg.norm(xg.astype(np.float64) - xo, axis=1)
    assert d.max() <= 1e-3 * R
    sim.close()


def test_explicit_interaction_matrix(B, orc):
    """PAPER.md:82 (Table 1, two-size run): a non-Berthelot eps matrix."""
    w = W.make_workload("C2", 8192)
    w.eps_matrix = 0.23 * np.array([[0.155, 1.26], [1.26, 0.155]])
    p = orc.params_from_workload(w)
    Fo, So, co, _ = orc.pair_forces(p, w.pos, w.type, "cells")
    sim = B.Simulation.from_workload(w)
    sim.compute_forces()
    Fg, cg = sim.get_forces()
    assert np.array_equal(cg, co)
    assert force_error(Fg, Fo, So) <= FORCE_TOL
    sim.close()


VARIANTS = [  # (sort, force kernel, tile sub-streams): lv_set_option; (0, 2) is the default path
    (1, 0, None), (1, 1, None), (1, 2, None), (0, 0, None), (0, 1, None), (0, 3, None), (1, 3, None),
    (0, 4, 1), (0, 4, 2), (0, 4, 4), (1, 4, 8), (0, 4, 16), (0, 4, 32),
]


@pytest.mark.parametrize("name,n,cpc", [("C1", None, None), ("C3", 20000, [1, 2, 2]),
                                         ("C4", 19999, [2]), ("C2", 8191, None)])
def test_implementation_options_do_not_change_results(B, orc, name, n, cpc):
    """lv_set_option: the multi-pass radix sort vs the one-digit (counting) sort
    and the four force kernels give bit-identical cell structures and neighbour
    counts, forces equal to rounding, and -- for the two sorts -- bit-identical
    trajectories."""
    w = workload(name, n)
    p = orc.params_from_workload(w)
    g = orc.grid_spec(p, cpc)
    key, ks, perm, off = orc.cell_structures(g, w.pos, w.type)
    Fo, So, co, _ = orc.pair_forces(p, w.pos, w.type, "cells")
    ref = B.Simulation.from_workload(w, cells_per_cut=cpc, neighbour_list=None)
    ref.compute_forces()
    F0, c0 = ref.get_forces()
    ref.step(30)
    x0, v0, _, _, _ = ref.get_state()
    ids0 = ref.get_debug(B.DBG_IDS_SORTED)
    ref.close()
    for sort, fk, sub in VARIANTS:
        opts = {B.OPT_SORT: sort, B.OPT_FORCE_KERNEL: fk}
        if sub is not None:
            opts[B.OPT_TILE_SUBSTREAMS] = sub
        sim = B.Simulation.from_workload(w, cells_per_cut=cpc, options=opts)
        sim.compute_forces()
        assert np.array_equal(sim.get_debug(B.DBG_KEYS), key)
        assert np.array_equal(sim.get_debug(B.DBG_KEYS_SORTED), ks)
        assert np.array_equal(sim.get_debug(B.DBG_PERM), perm)
        assert np.array_equal(sim.get_debug(B.DBG_CELL_OFFSETS), off)
        F, c = sim.get_forces()
        assert np.array_equal(c, co)
        assert force_error(F, Fo, So) <= FORCE_TOL
        assert force_error(F, F0.astype(np.float64), So) <= 2e-6
        sim.step(30)
        x, v, _, _, st = sim.get_state()
        assert st == 30
        if fk == 2:          # same force kernel as the default: the sort must not matter at all
            assert np.array_equal(x, x0) and np.array_equal(v, v0)
            assert np.array_equal(sim.get_debug(B.DBG_IDS_SORTED), ids0)
        else:
            R = w.R0
            assert np.abs(x.astype(np.float64) - x0).max() <= 1e-4 * R
        sim.close()
