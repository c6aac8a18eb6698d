"""Pins for the oracle's time step (steps (iii)-(vi)) and its
noise: closed forms of the linear recurrences, conservation laws, published
known answers.  CPU only."""
import os

import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def free_params(orc, a=1.0, b=0.0, **kw):
    """Non-interacting particles (eps = 0, q = 0), no wall unless asked."""
    d = dict(sigma=[1.0], mass=[1.0], charge=[0.0], wall_k=[0.0], drag_a=[a], kick_b=[b],
             dt=0.005, eps=[0.0], cut_factor=2.5, R0=1e9)
    d.update(kw)
    return orc.make_params(**d)


def far_lattice(N, spacing=200.0):
    """N distinct sites so far apart that no pair ever comes into range."""
    m = int(np.ceil(N ** (1.0 / 3.0)))
    g = (np.arange(m) - 0.5 * (m - 1)) * spacing
    return np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)[:N].copy()


# ---- Philox4x32-10 and the Gaussian kick ----------------------------------

def test_philox_known_answers(orc):
    rows = [l.split() for l in open(os.path.join(GOLD, "philox4x32_10_kat.txt"))
            if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(t, 16) for t in r]
        assert orc.philox4x32_10(v[0:4], v[4:6]) == v[6:10]


def test_gauss3_follows_box_muller_on_philox_words(orc):
    """u = ((w >> 9) + 0.5) 2^-23; (x, y) = sqrt(-2 ln u0) (cos, sin)(2 pi u1);
    z = sqrt(-2 ln u2) cos(2 pi u3); counter (id, n_lo, n_hi, 0), key = seed."""
    seed, pid, step = 0x0123456789ABCDEF, 77, (5 << 32) | 9
    w = orc.philox4x32_10([pid, 9, 5, 0], [seed & 0xFFFFFFFF, seed >> 32])
    u = [((x >> 9) + 0.5) / 2 ** 23 for x in w]
    xi = orc.gauss3(seed, [pid], step)[0]
    # invert Box-Muller instead of retyping it
    assert np.exp(-0.5 * (xi[0] ** 2 + xi[1] ** 2)) == pytest.approx(u[0], rel=1e-12)
    ang = np.arctan2(xi[1], xi[0]) / (2 * np.pi) % 1.0
    assert ang == pytest.approx(u[1], abs=1e-12)
    assert abs(xi[2]) <= np.sqrt(-2 * np.log(u[2])) * (1 + 1e-12)
    assert np.arccos(xi[2] / np.sqrt(-2 * np.log(u[2]))) / (2 * np.pi) == pytest.approx(
        min(u[3], 1 - u[3]), abs=1e-9)


def test_gauss3_moments_and_independence(orc):
    M = 200000
    xi = np.concatenate([orc.gauss3(42, np.arange(M // 4), s) for s in range(4)])
    for d in range(3):
        c = xi[:, d]
        assert abs(c.mean()) < 4 / np.sqrt(M)
        assert c.var() == pytest.approx(1.0, abs=4 * np.sqrt(2.0 / M))
        assert (c ** 4).mean() == pytest.approx(3.0, abs=4 * np.sqrt(96.0 / M))
    C = np.corrcoef(xi.T)
    assert np.max(np.abs(C - np.eye(3))) < 4 / np.sqrt(M)
    # different steps / ids / seeds give different draws; same inputs the same
    a = orc.gauss3(42, [5], 7)
    assert np.array_equal(a, orc.gauss3(42, [5], 7))
    assert not np.array_equal(a, orc.gauss3(42, [5], 8))
    assert not np.array_equal(a, orc.gauss3(42, [6], 7))
    assert not np.array_equal(a, orc.gauss3(43, [5], 7))


# ---- deterministic part of the update --------------------------------------

def test_free_flight_and_update_order(orc):
    """a = 1, b = 0, no force: v constant, x advances by dt v (semi-implicit
    Euler reduces to free flight)."""
    p = free_params(orc)
    x0 = np.array([[1.0, 2.0, 3.0]])
    v0 = np.array([[0.5, -1.0, 0.25]])
    x, v, bad = orc.step(p, x0, v0, [0], nsteps=10)
    assert bad == 0
    np.testing.assert_allclose(v, v0, rtol=0, atol=0)
    np.testing.assert_allclose(x, x0 + 10 * 0.005 * v0, rtol=1e-14)


def test_position_uses_new_velocity(orc):
    """DESIGN R16: x_{n+1} = x_n + dt v_{n+1}.  Under constant gravity from rest
    one step gives v = -g dt and x = -g dt^2 (explicit Euler would give x = 0)."""
    p = free_params(orc, g=2.0)
    x, v, _ = orc.step(p, np.zeros((1, 3)), np.zeros((1, 3)), [0], nsteps=1)
    assert v[0, 2] == pytest.approx(-2.0 * 0.005, rel=1e-14)
    assert x[0, 2] == pytest.approx(-2.0 * 0.005 ** 2, rel=1e-14)


def test_terminal_velocity_under_drag(orc):
    """v_{n+1} = a v_n - g dt  ->  v_inf = -g dt / (1 - a)  (= -g/gamma)."""
    a, b = orc.langevin_coeffs(1.0, 1.0, 1.0, 0.005)
    assert a == pytest.approx(0.995, rel=1e-15)
    assert b == pytest.approx(np.sqrt(1 - 0.995 ** 2), rel=1e-14)
    p = free_params(orc, a=a, g=0.3)
    x, v, _ = orc.step(p, np.zeros((1, 3)), np.zeros((1, 3)), [0], nsteps=6000)
    assert v[0, 2] == pytest.approx(-0.3 * 0.005 / (1 - a), rel=1e-9)
    assert v[0, 0] == 0.0


def test_wall_sees_new_radius(orc):
    """Steps (iii) before (iv), PAPER.md:66-67 (DESIGN R9): during step n the
    wall stands at R(n+1).  A particle at rest at |x| = R(0) - r: untouched if
    the wall stood at R(0), pushed by k (R(0) - R(1)) with R(1)."""
    p = free_params(orc, wall_k=[100.0], sched_mode=orc.SCHED_LINEAR, R0=20.0, R1=10.0,
                    sched_steps=100)
    x0 = np.array([[19.5, 0.0, 0.0]])
    x, v, _ = orc.step(p, x0, np.zeros((1, 3)), [0], step0=0, nsteps=1)
    assert v[0, 0] == pytest.approx(-0.005 * 100.0 * 0.1, rel=1e-12)
    # from step 50 the wall stands at R(51) = 14.9
    x, v, _ = orc.step(p, np.array([[14.5, 0.0, 0.0]]), np.zeros((1, 3)), [0], step0=50, nsteps=1)
    assert v[0, 0] == pytest.approx(-0.005 * 100.0 * 0.1, rel=1e-9)


def test_interface_drags_particle_at_steady_penetration(orc):
    """Linear interface at speed u with drag: steady pen = m gamma_eff u / k,
    from v = a v - (dt/m) k pen, v = -u/dt per step  ->  pen = (1-a) m u /(k dt^2)...
    written per step: u_step = (R0-R1)/S; pen = (1 - a) m u_step / (k dt^2)."""
    a = 0.9
    S = 200000
    p = free_params(orc, a=a, wall_k=[100.0], sched_mode=orc.SCHED_LINEAR, R0=20.0, R1=10.0,
                    sched_steps=S)
    u = 10.0 / S
    x, v, _ = orc.step(p, np.array([[19.5, 0.0, 0.0]]), np.zeros((1, 3)), [0], nsteps=4000)
    R_wall = orc.radius(p, 4000)           # wall position seen by the last step taken
    pen = x[0, 0] - (R_wall - 0.5)
    # the update reads x_n against R(n+1): subtract the one-step lag u
    assert pen + u == pytest.approx((1 - a) * u / (100.0 * 0.005 ** 2), rel=2e-3)


def test_energy_conservation_and_dt_scaling(orc):
    """Noise and drag off: total energy of a small LJ cluster (cut-off larger
    than the cluster, soft wall far away, gravity + centrifugal on) has no
    secular drift, and its fluctuation scales ~ dt (first-order symplectic)."""
    rng = np.random.default_rng(2)
    # 3x3x3 cubic cluster near the LJ minimum, small velocities
    g = np.arange(3) * 1.12
    x0 = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3) - 1.12
    v0 = rng.normal(0, 0.15, size=x0.shape)
    v0 -= v0.mean(axis=0)
    t = np.zeros(len(x0), dtype=np.int32)
    amps = []
    for dt, nsteps in ((0.002, 4000), (0.001, 8000)):
        p = orc.make_params(sigma=[1.0], mass=[1.0], charge=[0.0], wall_k=[100.0], drag_a=[1.0],
                            kick_b=[0.0], dt=dt, eps=[1.0], cut_factor=12.0, g=0.01,
                            omega2=(1e-3, 1e-3, 0.0), R0=2.6)
        x, v = x0.copy(), v0.copy()
        E = []
        for _ in range(40):
            x, v, bad = orc.step(p, x, v, t, nsteps=nsteps // 40, method="brute")
            assert bad == 0
            E.append(sum(orc.energy(p, 2.6, x, v, t)))
        E = np.array(E)
        E0 = sum(orc.energy(p, 2.6, x0, v0, t))
        slope = np.polyfit(np.arange(len(E)), E, 1)[0] * len(E)
        amps.append(np.std(E - E.mean()) + abs(E.mean() - E0))
        assert abs(slope) < 2e-3 * abs(E0)              # no secular drift
        assert np.max(np.abs(E - E0)) < 5e-3 * abs(E0)
    assert amps[1] < 0.75 * amps[0]                     # halving dt shrinks the error


def test_dimer_small_oscillation_period(orc):
    """Two unit masses at the LJ minimum: k = 72 eps / (2^(1/3) sigma^2) and
    reduced mass 1/2 give omega = 10.6908, period 0.58772 (textbook)."""
    dt = 0.0005
    p = orc.make_params(sigma=[1.0], mass=[1.0], charge=[0.0], wall_k=[0.0], drag_a=[1.0],
                        kick_b=[0.0], dt=dt, eps=[1.0], cut_factor=5.0, R0=1e9)
    r0 = 2.0 ** (1.0 / 6.0)
    x = np.array([[-(r0 + 0.002) / 2, 0, 0], [(r0 + 0.002) / 2, 0, 0]])
    v = np.zeros((2, 3))
    seps = []
    for _ in range(3000):
        x, v, _ = orc.step(p, x, v, [0, 0], nsteps=1, method="brute")
        seps.append(x[1, 0] - x[0, 0] - r0)
    s = np.array(seps)
    up = np.where((s[:-1] < 0) & (s[1:] >= 0))[0]
    period = np.mean(np.diff(up)) * dt
    assert period == pytest.approx(0.58772, rel=3e-3)


# ---- stochastic part: equipartition and Stokes-Einstein --------------------

def test_equipartition_and_msd_closed_form(orc):
    """Free particles: Var(v) obeys Var' = a^2 Var + b^2 -> kT/m exactly for
    b^2 = (kT/m)(1-a^2); MSD_1D(n) = dt^2 (kT/m) [ n(1+a)/(1-a)
    - 2a(1-a^n)/(1-a)^2 ]; long-time D = dt (kT/m)(1+a)/(2(1-a))."""
    N, dt, gamma, kT, m = 4096, 0.01, 2.0, 1.3, 2.0
    a, b = orc.langevin_coeffs(gamma, kT, m, dt)
    p = free_params(orc, a=a, b=b, dt=dt, mass=[m], seed=99)
    rng = np.random.default_rng(0)
    x0 = far_lattice(N)
    v0 = rng.normal(0, np.sqrt(kT / m), size=(N, 3))      # start in equilibrium
    t = np.zeros(N, dtype=np.int32)
    x, v = x0, v0
    ke, msd, ns = [], [], []
    n = 0
    for _ in range(8):
        x, v, bad = orc.step(p, x, v, t, step0=n, nsteps=200)
        n += 200
        ke.append(0.5 * m * (v ** 2).sum(axis=1).mean())
        msd.append(((x - x0) ** 2).mean())                 # per component
        ns.append(n)
    # equipartition: <1/2 m v^2> = 3/2 kT ; snapshots 2/gamma apart, ~independent
    se = 1.5 * kT * np.sqrt(2.0 / (3 * N * len(ke)))
    assert np.mean(ke) == pytest.approx(1.5 * kT, abs=4 * se)
    ns = np.array(ns, dtype=float)
    want = dt ** 2 * (kT / m) * (ns * (1 + a) / (1 - a) - 2 * a * (1 - a ** ns) / (1 - a) ** 2)
    # sampling error of a mean of 3N chi-square(1) variables
    np.testing.assert_allclose(msd, want, rtol=4 * np.sqrt(2.0 / (3 * N)))
    D = dt * (kT / m) * (1 + a) / (2 * (1 - a))
    assert D == pytest.approx(kT / (m * gamma) * (1 - gamma * dt / 2), rel=1e-12)
    # Stokes-Einstein: 3-D MSD = 6 D t at long time (t >> 1/gamma)
    slope = (msd[-1] - msd[3]) * 3 / ((ns[-1] - ns[3]) * dt)
    assert slope == pytest.approx(6 * D, rel=0.08)


def test_variance_recurrence_from_cold_start(orc):
    """Var_n = (kT/m)(1 - a^(2n)) from v = 0."""
    N, dt = 8192, 0.02
    a, b = orc.langevin_coeffs(1.0, 1.0, 1.0, dt)
    p = free_params(orc, a=a, b=b, dt=dt, seed=7)
    x, v, _ = orc.step(p, far_lattice(N), np.zeros((N, 3)), np.zeros(N, np.int32), nsteps=25)
    want = 1.0 - a ** 50
    assert v.var() == pytest.approx(want, rel=4 * np.sqrt(2.0 / (3 * N)))


def test_noise_keyed_on_id_and_step_split_invariance(orc):
    """lv_step(a); lv_step(b) == lv_step(a+b): the kick depends on (id, n) only."""
    N = 64
    a, b = orc.langevin_coeffs(1.0, 1.0, 1.0, 0.005)
    p = orc.make_params(sigma=[1.0], mass=[1.0], charge=[0.0], wall_k=[100.0], drag_a=[a],
                        kick_b=[b], dt=0.005, eps=[1.0], cut_factor=2.5, R0=6.0, seed=3)
    rng = np.random.default_rng(1)
    g = np.arange(4) * 1.3 - 1.95
    x0 = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)
    v0 = rng.normal(0, 1, size=(N, 3))
    t = np.zeros(N, np.int32)
    xa, va, _ = orc.step(p, x0, v0, t, step0=0, nsteps=30)
    xb, vb, _ = orc.step(p, x0, v0, t, step0=0, nsteps=12)
    xb, vb, _ = orc.step(p, xb, vb, t, step0=12, nsteps=18)
    assert np.array_equal(xa, xb) and np.array_equal(va, vb)
    xc, vc, _ = orc.step(p, x0, v0, t, step0=0, nsteps=30, method="brute")
    np.testing.assert_allclose(xc, xa, rtol=0, atol=1e-11)


def test_nonfinite_is_reported(orc):
    """DESIGN R6: coincident particles are not clamped; the step reports it."""
    p = orc.make_params(sigma=[1.0], mass=[1.0], charge=[0.0], wall_k=[0.0], drag_a=[1.0],
                        kick_b=[0.0], dt=0.005, eps=[1.0], R0=1e9)
    x = np.zeros((2, 3))
    _, _, bad = orc.step(p, x, np.zeros((2, 3)), [0, 0], nsteps=1, method="brute")
    assert bad == 1
