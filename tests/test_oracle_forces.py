"""Pins for the oracle's pair force (step (ii)) and surface /
external forces (steps (iv), (v)): closed forms, symmetry, and
the O(N^2) definition against the cell-list route.  CPU only."""
import numpy as np
import pytest

from paper_2501_04456_b200.workloads import make_workload, random_gas


def lj_params(orc, **kw):
    d = dict(sigma=[1.0], mass=[1.0], charge=[0.0], wall_k=[100.0], drag_a=[1.0],
             kick_b=[0.0], dt=0.005, eps=[1.0], cut_factor=2.5, R0=1e6)
    d.update(kw)
    return orc.make_params(**d)


def dimer(r):
    return np.array([[0.0, 0.0, 0.0], [r, 0.0, 0.0]])


# ---- LJ dimer closed forms (textbook 12-6; DESIGN R1) ---------------------

def test_lj_dimer_minimum(orc):
    p = lj_params(orc)
    F, S, cnt, U = orc.pair_forces(p, dimer(2.0 ** (1.0 / 6.0)), [0, 0], "brute")
    assert abs(F[1, 0]) < 1e-12 and abs(F[0, 0]) < 1e-12
    assert U == pytest.approx(-1.0, abs=1e-14)
    assert list(cnt) == [1, 1]


def test_lj_dimer_at_sigma_is_repulsive_24(orc):
    p = lj_params(orc)
    F, _, _, U = orc.pair_forces(p, dimer(1.0), [0, 0], "brute")
    assert F[1, 0] == pytest.approx(24.0, rel=1e-14)     # pushes particle 1 to +x
    assert F[0, 0] == pytest.approx(-24.0, rel=1e-14)
    assert abs(U) < 1e-14


def test_lj_truncated_not_shifted(orc):
    """range limited, values NOT shifted -> F and U jump at r_c."""
    p = lj_params(orc)
    F, _, cnt, U = orc.pair_forces(p, dimer(2.5 - 1e-6), [0, 0], "brute")
    assert F[1, 0] == pytest.approx(-0.0389995, rel=2e-5)  # attractive, not zero
    assert U == pytest.approx(-0.0163169, rel=2e-5)
    assert list(cnt) == [1, 1]
    for r in (2.5, 2.5 + 1e-3, 7.0):                       # zero at and beyond
        F, _, cnt, U = orc.pair_forces(p, dimer(r), [0, 0], "brute")
        assert np.all(F == 0.0) and U == 0.0 and list(cnt) == [0, 0]


def test_lj_scales_with_eps_and_sigma(orc):
    p = lj_params(orc, sigma=[1.7], eps=[3.0])
    rmin = 2.0 ** (1.0 / 6.0) * 1.7
    F, _, _, U = orc.pair_forces(p, dimer(rmin), [0, 0], "brute")
    assert abs(F[1, 0]) < 1e-11 and U == pytest.approx(-3.0, rel=1e-13)
    F, _, _, _ = orc.pair_forces(p, dimer(1.7), [0, 0], "brute")
    assert F[1, 0] == pytest.approx(24.0 * 3.0 / 1.7, rel=1e-13)


# ---- Coulomb closed form (DESIGN R5) --------------------------------------

def test_coulomb_closed_form(orc):
    # eps = 0 isolates the Coulomb term; l_B = 0.7, unit charges, cut 5 sigma
    p = lj_params(orc, sigma=[1.0, 1.0], mass=[1.0] * 2, charge=[1.0, -1.0], wall_k=[0.0] * 2,
                  drag_a=[1.0] * 2, kick_b=[0.0] * 2, eps=[0.0, 0.0], cut_factor=5.0,
                  coulomb_k=0.7)
    for r in (0.8, 1.0, 3.3):
        F, _, _, U = orc.pair_forces(p, dimer(r), [0, 0], "brute")       # like charges
        assert F[1, 0] == pytest.approx(0.7 / r ** 2, rel=1e-13)          # repulsive
        assert U == pytest.approx(0.7 / r, rel=1e-13)
        F, _, _, U = orc.pair_forces(p, dimer(r), [0, 1], "brute")       # unlike
        assert F[1, 0] == pytest.approx(-0.7 / r ** 2, rel=1e-13)         # attractive
        assert U == pytest.approx(-0.7 / r, rel=1e-13)
    F, _, _, _ = orc.pair_forces(p, dimer(5.0 - 1e-6), [0, 0], "brute")
    assert F[1, 0] == pytest.approx(0.028, rel=1e-5)                      # unshifted jump
    F, _, _, U = orc.pair_forces(p, dimer(5.0), [0, 0], "brute")
    assert np.all(F == 0.0) and U == 0.0


def test_force_direction_is_along_separation(orc):
    p = lj_params(orc)
    x = np.array([[0.3, -0.2, 0.5], [1.0, 0.6, -0.1]])
    F, _, _, _ = orc.pair_forces(p, x, [0, 0], "brute")
    d = x[1] - x[0]
    assert np.linalg.norm(np.cross(F[1], d)) < 1e-14
    r = np.linalg.norm(d)
    fmag = 24.0 * (2.0 / r ** 12 - 1.0 / r ** 6) / r
    assert np.dot(F[1], d) / r == pytest.approx(fmag, rel=1e-13)


# ---- mixing rules (PAPER.md:64 r_A + r_B; DESIGN R2-R4) -------------------

def test_lorentz_berthelot_tables(orc):
    w = make_workload("C2", state=False)
    p = orc.params_from_workload(w)
    M = orc.MAX_TYPES
    assert p.sig[0 * M + 1] == pytest.approx(1.25) and p.sig[1 * M + 0] == pytest.approx(1.25)
    assert p.sig[1 * M + 1] == pytest.approx(1.5)
    assert p.eps[0 * M + 1] == pytest.approx(np.sqrt(2.0))
    assert p.rcut[0 * M + 0] == pytest.approx(5.0)
    assert p.rcut[0 * M + 1] == pytest.approx(6.25)
    assert p.rcut[1 * M + 1] == pytest.approx(7.5)


def test_per_pair_cutoff_is_used(orc):
    w = make_workload("C2", state=False)
    p = orc.params_from_workload(w)
    # r = 6.0: inside r_c(0,1) = 6.25 and r_c(1,1) = 7.5, outside r_c(0,0) = 5
    assert list(orc.pair_forces(p, dimer(6.0), [0, 0], "brute")[2]) == [0, 0]
    assert list(orc.pair_forces(p, dimer(6.0), [0, 1], "brute")[2]) == [1, 1]
    assert list(orc.pair_forces(p, dimer(7.0), [0, 1], "brute")[2]) == [0, 0]
    assert list(orc.pair_forces(p, dimer(7.0), [1, 1], "brute")[2]) == [1, 1]


# ---- definition (brute) vs cell list; Newton III; F = -grad U -------------

def _mixed_params(orc, T):
    sig = [1.0, 1.5, 2.5][:T]
    return orc.make_params(sigma=sig, mass=[s ** 3 for s in sig], charge=[0.0, 1.0, -1.0][:T],
                           wall_k=[100.0] * T, drag_a=[1.0] * T, kick_b=[0.0] * T, dt=0.002,
                           eps=[1.0, 3.0, 0.5][:T], cut_factor=3.0, coulomb_k=0.7, R0=1e6)


@pytest.mark.parametrize("T,n,box", [(1, 1500, 14.0), (2, 2500, 22.0), (3, 4096, 34.0)])
def test_cells_equal_brute_uniform(orc, T, n, box):
    p = _mixed_params(orc, T)
    x, t = random_gas(n, T, box, seed=10 + T, min_sep=0.8)
    Fb, Sb, cb, Ub = orc.pair_forces(p, x, t, "brute")
    Fc, Sc, cc, Uc = orc.pair_forces(p, x, t, "cells")
    assert np.array_equal(cb, cc)
    assert cb.sum() > 10 * len(t)
    assert np.max(np.abs(Fb - Fc) / Sb[:, None].clip(1e-300)) < 1e-12
    assert Uc == pytest.approx(Ub, rel=1e-11)
    np.testing.assert_allclose(Sc, Sb, rtol=1e-12)


def test_cells_equal_brute_clustered(orc):
    """Clustered input: a few dense blobs far apart (crowded and empty cells)."""
    p = _mixed_params(orc, 3)
    rng = np.random.default_rng(5)
    centres = rng.uniform(-60, 60, size=(6, 3))
    x = (centres[rng.integers(0, 6, 3000)] + rng.normal(0, 2.5, size=(3000, 3))).astype(np.float32)
    t = rng.integers(0, 3, 3000).astype(np.int32)
    Fb, Sb, cb, _ = orc.pair_forces(p, x, t, "brute")
    Fc, _, cc, _ = orc.pair_forces(p, x, t, "cells")
    assert np.array_equal(cb, cc)
    assert np.max(np.abs(Fb - Fc) / Sb[:, None].clip(1e-300)) < 1e-12


def test_newton_third_law(orc):
    p = _mixed_params(orc, 3)
    x, t = random_gas(3000, 3, 30.0, seed=3, min_sep=0.8)
    F, S, _, _ = orc.pair_forces(p, x, t, "cells")
    assert np.all(np.abs(F.sum(axis=0)) <= 1e-10 * S.sum())
    # and zero net torque (central forces)
    assert np.all(np.abs(np.cross(x.astype(np.float64), F).sum(axis=0)) <= 1e-9 * (S.sum() * 30))


def test_force_is_minus_gradient_of_energy(orc):
    """Central finite difference of the returned pair energy; the cluster is
    smaller than every cut-off so no pair crosses r_c (unshifted jump)."""
    p = _mixed_params(orc, 3)
    rng = np.random.default_rng(11)
    x = rng.uniform(-1.6, 1.6, size=(14, 3))
    x = x[[i for i in range(14) if all(np.linalg.norm(x[i] - x[j]) > 0.9 for j in range(i))]]
    t = (np.arange(len(x)) % 3).astype(np.int32)
    F, _, cnt, _ = orc.pair_forces(p, x, t, "brute")
    assert np.all(cnt == len(x) - 1)
    h = 1e-5
    for i in range(len(x)):
        for d in range(3):
            xp, xm = x.copy(), x.copy()
            xp[i, d] += h
            xm[i, d] -= h
            g = (orc.pair_forces(p, xp, t, "brute")[3] - orc.pair_forces(p, xm, t, "brute")[3]) / (2 * h)
            assert F[i, d] == pytest.approx(-g, rel=2e-6, abs=1e-6)


def test_S_is_sum_of_term_magnitudes(orc):
    p = _mixed_params(orc, 2)
    r = 1.3
    F, S, _, _ = orc.pair_forces(p, dimer(r), [1, 1], "brute")
    eps, sig, qq = 3.0, 1.5, 0.7
    s6 = (sig / r) ** 6
    assert S[0] == pytest.approx(48 * eps * s6 * s6 / r + 24 * eps * s6 / r + qq / r ** 2, rel=1e-13)


def test_in_range_predicate_is_fp32(orc):
    """DESIGN fp32 contract #2: the decision r^2 < r_c^2 is taken in fp32 on
    the fp32 state -- a pair whose fp64 distance is inside r_c by less than
    fp32 resolution must be decided by the fp32 expression."""
    p = lj_params(orc)
    rc2 = np.float32(2.5 * 2.5)
    below = np.nextafter(np.float32(2.5), np.float32(0))          # fp32 just below 2.5
    for r in (below, np.float32(2.5)):
        r2 = np.float32(r) * np.float32(r)                         # fl32(dx*dx), dy = dz = 0
        expect = int(r2 < rc2)
        cnt = orc.pair_forces(p, dimer(float(r)), [0, 0], "brute")[2]
        assert list(cnt) == [expect, expect]


# ---- surface spring and external forces ------------------------------------

def ext_params(orc, **kw):
    d = dict(sigma=[1.0, 2.0], mass=[1.0, 8.0], charge=[0.0, 0.0], wall_k=[100.0, 40.0],
             drag_a=[1.0, 1.0], kick_b=[0.0, 0.0], dt=0.005, eps=[1.0, 1.0], R0=20.0)
    d.update(kw)
    return orc.make_params(**d)


def test_wall_zero_inside_and_equilibrium_one_radius_inside(orc):
    """spring equilibrium 'at the distance of an NP radius from the surface'."""
    p = ext_params(orc)
    x = np.array([[0, 0, 0], [19.5, 0, 0], [0, -19.0, 0], [0, 0, 19.0]], dtype=float)
    F, S, U = orc.external_forces(p, 20.0, x, [0, 0, 1, 1])
    assert np.all(F == 0.0) and U == 0.0


def test_wall_harmonic_radial_inward(orc):
    p = ext_params(orc)
    d = np.array([1.0, 2.0, -2.0]) / 3.0
    x = (19.5 + 0.25) * d[None, :]
    F, S, U = orc.external_forces(p, 20.0, x, [0])
    np.testing.assert_allclose(F[0], -100.0 * 0.25 * d, rtol=1e-12)
    assert U == pytest.approx(0.5 * 100.0 * 0.25 ** 2, rel=1e-12)
    x = (19.0 + 0.5) * d[None, :]                     # type 1: r = 1, k = 40
    F, _, _ = orc.external_forces(p, 20.0, x, [1])
    np.testing.assert_allclose(F[0], -40.0 * 0.5 * d, rtol=1e-12)


def test_wall_window_mode(orc):
    """NPs in the range (-r_NP, r_NP) from the surface."""
    p = ext_params(orc, wall_mode=orc.WALL_WINDOW)
    for r, on in ((19.4, False), (19.6, True), (20.4, True), (20.6, False)):
        F, _, _ = orc.external_forces(p, 20.0, np.array([[r, 0.0, 0.0]]), [0])
        assert (F[0, 0] != 0.0) == on
    p = ext_params(orc)                                # one-sided: never lets go
    F, _, _ = orc.external_forces(p, 20.0, np.array([[25.0, 0.0, 0.0]]), [0])
    assert F[0, 0] == pytest.approx(-100.0 * 5.5)


def test_gravity_and_centrifugal(orc):
    p = ext_params(orc, wall_k=[0.0, 0.0], g=0.01, omega2=(4e-4, 4e-4, 0.0))
    x = np.array([[3.0, -2.0, 5.0], [1.0, 1.0, 1.0]])
    F, S, U = orc.external_forces(p, 20.0, x, [0, 1])
    np.testing.assert_allclose(F[0], [4e-4 * 3.0, -4e-4 * 2.0, -0.01], rtol=1e-13)
    np.testing.assert_allclose(F[1], [8 * 4e-4, 8 * 4e-4, -8 * 0.01], rtol=1e-13)
    assert U == pytest.approx(0.01 * 5 + 8 * 0.01 * 1 - 0.5 * 4e-4 * (9 + 4) - 0.5 * 8 * 4e-4 * 2)


def test_static_balances(orc):
    """Closed-form equilibria: gravity pen = m g / k; centrifugal
    rho_eq = k (R - r) / (k - m W^2)."""
    R, k, m, r = 20.0, 100.0, 1.0, 0.5
    p = ext_params(orc, g=0.3)
    pen = m * 0.3 / k
    F, _, _ = orc.external_forces(p, R, np.array([[0.0, 0.0, -(R - r + pen)]]), [0])
    assert abs(F[0, 2]) < 1e-12
    W2 = 2.0
    p = ext_params(orc, omega2=(W2, W2, W2))
    rho = k * (R - r) / (k - m * W2)
    F, _, _ = orc.external_forces(p, R, np.array([[rho, 0.0, 0.0]]), [0])
    assert abs(F[0, 0]) < 1e-11


# ---- schedule (step (iii); radius-square law PAPER.md:58) -----

def test_schedule_closed_forms(orc):
    p = ext_params(orc, sched_mode=orc.SCHED_LINEAR, R0=60.0, R1=25.0, sched_steps=10000)
    assert orc.radius(p, 0) == 60.0
    assert orc.radius(p, 10000) == 25.0
    assert orc.radius(p, 123456) == 25.0
    assert orc.radius(p, 2500) == pytest.approx(60.0 - 35.0 * 0.25, rel=1e-15)
    p = ext_params(orc, sched_mode=orc.SCHED_R2LAW, R0=60.0, R1=25.0, sched_steps=10000)
    n = np.array([0, 1000, 5000, 9999, 10000])
    R2 = np.array([orc.radius(p, int(k)) ** 2 for k in n])
    np.testing.assert_allclose(np.diff(R2) / np.diff(n), (25.0 ** 2 - 60.0 ** 2) / 10000, rtol=1e-11)
    assert orc.radius(p, 10000) == 25.0
    p = ext_params(orc, sched_mode=orc.SCHED_LINEAR, R0=10.0, R1=30.0, sched_steps=100)
    assert orc.radius(p, 50) == pytest.approx(20.0)      # condensation
    p = ext_params(orc, sched_mode=orc.SCHED_CONST, R0=20.0, R1=5.0, sched_steps=100)
    assert orc.radius(p, 50) == 20.0
