"""Seeded synthetic inputs: BASELINE.json's five configurations and scaled-down
copies of them.  NEUTRAL MODULE: it serves both the CUDA path and the test
oracle, and holds none of the method's arithmetic -- no forces, no mixing
rules, no Langevin coefficients, no grid, no noise.  It produces physical
parameters in reduced units plus fp32 initial positions / velocities / types;
each side derives its own tables from them.

The inputs are synthetic stand-ins for the paper's workloads (10^4 NPs of
r = 0.5 um in R0 = 20 um; 39 500 + 1 500 NPs of two sizes in a
drying droplet; "up to 2.5 x 10^5" NPs).  The
paper's own parameter files and frames (ref [55]) are not here
and are not needed.  Recipe:
  * NPs "randomly distributed in a sphere": uniform in the ball
    |x| <= R0 - r_a, rejected to a minimum separation 0.9 sigma_ab, largest
    type first;
  * Maxwell-Boltzmann velocities, variance kT/m_a per component;
  * type counts round(f N), the last type takes the remainder, ids blockwise
    by type;  m_a = (sigma_a/sigma_0)^3 (equal material density);
  * C4: FCC lattice clipped to the ball, jittered by +-0.05 sigma.
Generator RNG: numpy PCG64 seeded with the configuration's seed.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import List, Optional, Sequence

import numpy as np

SCHED_CONST, SCHED_LINEAR, SCHED_R2LAW = 0, 1, 2
WALL_ONESIDED, WALL_WINDOW = 0, 1


@dataclass
class Workload:
    name: str
    n: int
    sigma: List[float]          # NP diameters (r_NP = sigma/2)
    eps: List[float]            # per-type LJ well depth (Berthelot-mixed by each side)
    charge: List[float]
    mass: List[float]
    wall_k: List[float]         # surface spring constant per type
    gamma: List[float]          # velocity relaxation rate per type
    fractions: List[float]
    kT: float
    dt: float
    cut_factor: float           # r_c,ab = cut_factor * sigma_ab
    coulomb_k: float            # Bjerrum length * kT
    g: float
    omega2: Sequence[float]
    wall_mode: int
    sched_mode: int
    R0: float
    R1: float
    sched_steps: int
    seed: int
    steps: int
    init: str                   # "ball" | "fcc"
    eps_matrix: Optional[np.ndarray] = None
    pos: np.ndarray = field(default=None, repr=False)    # [n,3] float32
    vel: np.ndarray = field(default=None, repr=False)    # [n,3] float32
    type: np.ndarray = field(default=None, repr=False)   # [n] int32

    @property
    def n_types(self) -> int:
        return len(self.sigma)


def _mass(sigma):
    return [(s / sigma[0]) ** 3 for s in sigma]


def _spec(name: str) -> Workload:
    """BASELINE.json configs[0..4] with the readings of DESIGN.md."""
    if name == "C1":
        s = [1.0]
        return Workload("C1", 2048, s, [1.0], [0.0], _mass(s), [100.0], [1.0], [1.0],
                        kT=1.0, dt=0.005, cut_factor=2.5, coulomb_k=0.0, g=0.0,
                        omega2=(0.0, 0.0, 0.0), wall_mode=WALL_ONESIDED,
                        sched_mode=SCHED_CONST, R0=20.0, R1=20.0, sched_steps=0,
                        seed=1, steps=1000, init="ball")
    if name == "C2":
        s = [1.0, 1.5]
        return Workload("C2", 32768, s, [1.0, 2.0], [1.0, -1.0], _mass(s), [100.0] * 2,
                        [1.0] * 2, [0.7, 0.3], kT=1.0, dt=0.002, cut_factor=5.0,
                        coulomb_k=0.7, g=0.0, omega2=(0.0, 0.0, 0.0),
                        wall_mode=WALL_ONESIDED, sched_mode=SCHED_LINEAR, R0=60.0, R1=25.0,
                        sched_steps=10000, seed=2, steps=10000, init="ball")
    if name == "C3":
        s = [1.0, 1.5, 2.5]
        w2 = 0.005 ** 2
        return Workload("C3", 250000, s, [1.0, 3.0, 0.5], [0.0, 1.0, -1.0], _mass(s),
                        [100.0] * 3, [2.0] * 3, [0.5, 0.3, 0.2], kT=1.0, dt=0.002,
                        cut_factor=5.0, coulomb_k=0.7, g=0.01, omega2=(w2, w2, 0.0),
                        wall_mode=WALL_ONESIDED, sched_mode=SCHED_LINEAR, R0=150.0, R1=50.0,
                        sched_steps=20000, seed=3, steps=20000, init="ball")
    if name == "C4":
        s = [1.0]
        n = 250000
        R = (n * 0.125 / 0.40) ** (1.0 / 3.0)
        return Workload("C4", n, s, [10.0], [0.0], _mass(s), [100.0], [1.0], [1.0],
                        kT=0.5, dt=0.001, cut_factor=2.5, coulomb_k=0.0, g=0.0,
                        omega2=(0.0, 0.0, 0.0), wall_mode=WALL_ONESIDED,
                        sched_mode=SCHED_CONST, R0=R, R1=R, sched_steps=0,
                        seed=4, steps=5000, init="fcc")
    if name == "C5":
        s = [1.0, 1.2]
        return Workload("C5", 1048576, s, [1.0, 1.0], [0.5, -0.5], _mass(s), [100.0] * 2,
                        [1.0] * 2, [0.5, 0.5], kT=1.0, dt=0.002, cut_factor=4.0,
                        coulomb_k=0.7, g=0.0, omega2=(0.0, 0.0, 0.0),
                        wall_mode=WALL_ONESIDED, sched_mode=SCHED_LINEAR, R0=250.0, R1=120.0,
                        sched_steps=10000, seed=5, steps=10000, init="ball")
    # ---- paper-shaped scenarios (Table 1) in reduced units; synthetic
    # stand-ins: the authors' parameter files are not available
    if name == "T8":
        # edge case, not a BASELINE config: the maximum number of coexisting types (T = 8 =
        # LV_MAX_TYPES), eight sizes, alternating charges, every force term switched on
        s = [1.0, 1.2, 1.4, 1.6, 1.8, 2.0, 2.2, 2.4]
        return Workload("T8", 12000, s, [1.0, 2.0, 0.5, 1.5, 3.0, 0.7, 1.2, 2.5],
                        [0.0, 1.0, -1.0, 0.5, -0.5, 0.0, 2.0, -2.0], _mass(s), [100.0] * 8, [1.5] * 8,
                        [0.2, 0.15, 0.15, 0.1, 0.1, 0.1, 0.1, 0.1], kT=1.0, dt=0.002, cut_factor=3.0,
                        coulomb_k=0.7, g=0.01, omega2=(2.5e-5, 2.5e-5, 0.0), wall_mode=WALL_ONESIDED,
                        sched_mode=SCHED_LINEAR, R0=45.0, R1=25.0, sched_steps=5000, seed=21,
                        steps=5000, init="ball")
    if name == "P1":
        # row "1" (Fig. 2, 7): R0 = 20 um, r_NP = 0.5 um -> sigma = 1, R0 = 20; 10^4 neutral NPs,
        # LJ only, range 4 (r_A + r_B), no evaporation, random tumbling =
        # isotropic centrifugal force; the paper's windowed surface force
        s = [1.0]
        w2 = 0.05 ** 2
        return Workload("P1", 10000, s, [1.0], [0.0], _mass(s), [100.0], [1.0], [1.0],
                        kT=1.0, dt=0.005, cut_factor=4.0, coulomb_k=0.0, g=0.0,
                        omega2=(w2, w2, w2), wall_mode=WALL_WINDOW,
                        sched_mode=SCHED_CONST, R0=20.0, R1=20.0, sched_steps=0,
                        seed=11, steps=5000, init="ball")
    if name == "P8":
        # row "8" (Fig. 8, 9): R0 = 60 um, r_NP = 0.25 / 1.5 um (6 : 1) -> sigma = 1 / 6,
        # R0 = 120; 39 500 + 1 500 neutral NPs; eps = 0.23 [[0.155, 0.155], [0, 1.26]] is not a
        # Berthelot matrix (and prints a 0 below the diagonal: read as symmetric), here in units
        # of eps_11; radius-square-law evaporation until nearly dry; rotation
        # about one axis
        s = [1.0, 6.0]
        w2 = 0.01 ** 2
        eps = np.array([[1.0, 1.0], [1.0, 1.26 / 0.155]])
        return Workload("P8", 41000, s, [1.0, 1.26 / 0.155], [0.0, 0.0], _mass(s), [100.0] * 2,
                        [1.0] * 2, [39500.0 / 41000.0, 1500.0 / 41000.0], kT=1.0, dt=0.002,
                        cut_factor=4.0, coulomb_k=0.0, g=0.0, omega2=(w2, w2, 0.0),
                        wall_mode=WALL_ONESIDED, sched_mode=SCHED_R2LAW, R0=120.0, R1=48.0,
                        sched_steps=20000, seed=18, steps=20000, init="ball", eps_matrix=eps)
    raise KeyError(name)


def type_counts(n: int, fractions: Sequence[float]) -> List[int]:
    counts = [int(round(f * n)) for f in fractions[:-1]]
    counts.append(n - sum(counts))
    assert min(counts) >= 0
    return counts


def _ball_points(rng, m, radius):
    d = rng.standard_normal((m, 3))
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    r = radius * rng.random(m) ** (1.0 / 3.0)
    return d * r[:, None]


def ball_min_separation(rng, counts, sigma, R0, sep_factor=0.9):
    """Uniform points in the ball |x| <= R0 - r_a with pair separation
    >= sep_factor * sigma_ab, inserted largest type first in batches (a batch
    member is dropped if it conflicts with an accepted point or with an
    earlier member of its batch)."""
    from scipy.spatial import cKDTree

    T = len(counts)
    out = [np.zeros((0, 3)) for _ in range(T)]
    order = sorted(range(T), key=lambda a: -sigma[a])
    for a in order:
        need = counts[a]
        guard = 0
        while need > 0:
            guard += 1
            if guard > 10000:
                raise RuntimeError("rejection sampling does not converge (too dense)")
            m = int(need * 1.25) + 16
            cand = _ball_points(rng, m, R0 - 0.5 * sigma[a])
            ok = np.ones(m, dtype=bool)
            for b in range(T):
                if out[b].shape[0] == 0:
                    continue
                rab = sep_factor * 0.5 * (sigma[a] + sigma[b])
                cnt = cKDTree(out[b]).query_ball_point(cand, rab, return_length=True)
                ok &= cnt == 0
            cand = cand[ok]
            if cand.shape[0] > 1:
                pairs = cKDTree(cand).query_pairs(sep_factor * sigma[a], output_type="ndarray")
                if pairs.size:
                    drop = np.zeros(cand.shape[0], dtype=bool)
                    drop[pairs.max(axis=1)] = True
                    cand = cand[~drop]
            cand = cand[:need]
            out[a] = np.concatenate([out[a], cand], axis=0)
            need -= cand.shape[0]
    return np.concatenate(out, axis=0)


def fcc_ball(rng, n, sigma, R, jitter=0.05):
    """FCC sites with |x| <= R - sigma/2, lattice constant bisected so that at
    least n sites fit, surplus outermost sites dropped (ties by index),
    jittered uniformly by +-jitter per coordinate."""
    rin = R - 0.5 * sigma
    basis = np.array([[0, 0, 0], [0.5, 0.5, 0], [0.5, 0, 0.5], [0, 0.5, 0.5]])

    def sites(a):
        m = int(np.ceil(rin / a)) + 1
        k = np.arange(-m, m + 1)
        gx, gy, gz = np.meshgrid(k, k, k, indexing="ij")
        cells = np.stack([gx.ravel(), gy.ravel(), gz.ravel()], axis=1).astype(np.float64)
        pts = (cells[:, None, :] + basis[None, :, :]).reshape(-1, 3) * a
        r2 = (pts ** 2).sum(axis=1)
        keep = r2 <= rin * rin
        return pts[keep], r2[keep]

    lo, hi = 0.5 * sigma, 4.0 * sigma * max(1.0, (rin ** 3 / n) ** (1.0 / 3.0))
    for _ in range(40):
        mid = 0.5 * (lo + hi)
        if sites(mid)[0].shape[0] >= n:
            lo = mid
        else:
            hi = mid
    pts, r2 = sites(lo)
    order = np.argsort(r2, kind="stable")[:n]
    order.sort()
    pts = pts[order]
    pts += rng.uniform(-jitter, jitter, size=pts.shape)
    return pts


def make_workload(name: str, n: Optional[int] = None, state: bool = True,
                  seed: Optional[int] = None) -> Workload:
    """BASELINE config `name` ("C1".."C5"), paper-shaped scenario ("P1", "P8") or the eight-type edge case ("T8").  With n given, a scaled-down (or
    up) copy at the same volume fractions: radii scale as (n/N)^(1/3).  `seed`
    overrides the configuration's seed (independent replicas)."""
    w = _spec(name)
    if seed is not None:
        w = replace(w, seed=int(seed))
    if n is not None and n != w.n:
        f = (n / w.n) ** (1.0 / 3.0)
        w = replace(w, n=n, R0=w.R0 * f, R1=w.R1 * f, name=f"{w.name}@{n}")
    if not state:
        return w
    rng = np.random.Generator(np.random.PCG64(w.seed))
    counts = type_counts(w.n, w.fractions)
    typ = np.repeat(np.arange(w.n_types, dtype=np.int32), counts)
    if w.init == "ball":
        pos = ball_min_separation(rng, counts, w.sigma, w.R0)
    else:
        pos = fcc_ball(rng, w.n, w.sigma[0], w.R0)
    std = np.sqrt(w.kT / np.asarray(w.mass))[typ]
    vel = rng.standard_normal((w.n, 3)) * std[:, None]
    w.pos = np.ascontiguousarray(pos, dtype=np.float32)
    w.vel = np.ascontiguousarray(vel, dtype=np.float32)
    w.type = typ
    return w


def random_gas(n, n_types, box, seed, sigma=None, min_sep=0.0):
    """Small helper for tests: n points uniform in a cube of edge `box`
    centred at the origin, types uniform at random; fp32."""
    rng = np.random.Generator(np.random.PCG64(seed))
    pos = rng.uniform(-0.5 * box, 0.5 * box, size=(n, 3))
    typ = rng.integers(0, n_types, size=n).astype(np.int32)
    if min_sep > 0 and n > 1:
        from scipy.spatial import cKDTree
        pairs = cKDTree(pos).query_pairs(min_sep, output_type="ndarray")
        if pairs.size:
            keep = np.ones(n, dtype=bool)
            keep[pairs.max(axis=1)] = False
            pos, typ = pos[keep], typ[keep]
    return np.ascontiguousarray(pos, dtype=np.float32), typ
