"""Pins for the oracle's cell structures (step (i)) -- the fp32
contracts the CUDA path must reproduce bit for bit -- and for the input
generators.  Invariants and geometric properties, not a retyped formula.
CPU only."""
import numpy as np
import pytest

from paper_2501_04456_b200.workloads import make_workload, type_counts


@pytest.fixture(scope="module")
def c2small():
    return make_workload("C2", n=4096)


def decode(g, key, typ):
    base = np.array([g.base[b] for b in range(g.n_types)], dtype=np.int64)[typ]
    G = np.array([g.G[b] for b in range(g.n_types)], dtype=np.int64)[typ]
    c = key.astype(np.int64) - base
    return np.stack([c % G, (c // G) % G, c // (G * G)], axis=1), G


@pytest.mark.parametrize("cpc", [None, [1, 1], [2, 3]])
def test_cell_keys_geometry(orc, c2small, cpc):
    """A key decodes to the cell that contains the particle (to fp32 rounding
    of one cell coordinate), on the grid of the particle's own type, and key
    ranges of different types do not overlap."""
    w = c2small
    p = orc.params_from_workload(w)
    g = orc.grid_spec(p, cpc)
    key, ks, perm, off = orc.cell_structures(g, w.pos, w.type)
    c, G = decode(g, key, w.type)
    assert np.all(c >= 0) and np.all(c < G[:, None])
    for b in range(g.n_types):
        m = w.type == b
        assert np.all(key[m] >= g.base[b]) and np.all(key[m] < g.base[b + 1])
    h = np.array([g.h[b] for b in range(g.n_types)])[w.type]
    lo = -0.5 * G * h
    t = (w.pos.astype(np.float64) - lo[:, None]) / h[:, None]
    assert np.all(np.abs(np.floor(t) - c) <= 1)
    assert np.mean(np.floor(t) == c) > 0.999            # off by one only at a cell face
    assert np.all(np.abs(t - (c + 0.5)) <= 0.5 + 1e-4)


def test_grid_rule(orc, c2small):
    """DESIGN 'Grid rule': h_b = r_c,bb (1 + 2^-9) / k_b, the grid covers the
    largest droplet plus one largest NP diameter, w_ab cells reach r_c,ab."""
    w = c2small
    p = orc.params_from_workload(w)
    M = orc.MAX_TYPES
    for cpc in ([1, 1], [2, 3]):
        g = orc.grid_spec(p, cpc)
        for b in range(2):
            assert g.h[b] == pytest.approx(p.rcut[b * M + b] * (1 + 2.0 ** -9) / cpc[b], rel=1e-15)
            assert g.G[b] * g.h[b] >= 2 * max(w.R0, w.R1) + 2 * max(w.sigma)
            assert (g.G[b] - 1) * g.h[b] < 2 * max(w.R0, w.R1) + 2 * max(w.sigma)
            assert g.lo[b] == np.float32(-0.5 * g.G[b] * g.h[b])
            assert g.inv_h[b] == np.float32(1.0 / g.h[b])
            for a in range(2):
                assert g.w[a * M + b] * g.h[b] >= p.rcut[a * M + b] * (1 + 2.0 ** -10)
                assert (g.w[a * M + b] - 1) * g.h[b] < p.rcut[a * M + b] * (1 + 2.0 ** -10)
        assert g.base[0] == 0 and g.base[1] == g.G[0] ** 3
        assert g.base[2] == g.G[0] ** 3 + g.G[1] ** 3


@pytest.mark.parametrize("cpc", [None, [2, 3]])
def test_every_in_range_pair_is_inside_the_stencil(orc, c2small, cpc):
    """What the grid is for: any pair the fp32 predicate accepts
    lies within w_ab cells per axis on the grid of the neighbour's type."""
    from scipy.spatial import cKDTree
    w = c2small
    p = orc.params_from_workload(w)
    g = orc.grid_spec(p, cpc)
    M = orc.MAX_TYPES
    x = w.pos.astype(np.float64)
    pairs = cKDTree(x).query_pairs(7.6, output_type="ndarray")
    i = np.concatenate([pairs[:, 0], pairs[:, 1]])
    j = np.concatenate([pairs[:, 1], pairs[:, 0]])
    rc = np.array([[p.rcut[a * M + b] for b in range(2)] for a in range(2)])[w.type[i], w.type[j]]
    d = np.linalg.norm(x[i] - x[j], axis=1)
    m = d < rc * (1 + 1e-6)
    i, j = i[m], j[m]
    assert len(i) > 20000
    # cell of target i on the grid of j's type, cell of j on its own grid
    for b in range(2):
        sel = w.type[j] == b
        ii, jj = i[sel], j[sel]
        tb = np.full(w.n, b, dtype=np.int32)
        kb = orc.cell_structures(g, w.pos, tb)[0]           # everyone binned on grid b
        cb, _ = decode(g, kb, tb)
        wab = np.array([g.w[a * M + b] for a in range(2)])[w.type[ii]]
        assert np.all(np.abs(cb[ii] - cb[jj]).max(axis=1) <= wab)


def test_sort_is_stable_and_a_permutation(orc, c2small):
    w = c2small
    p = orc.params_from_workload(w)
    g = orc.grid_spec(p)
    key, ks, perm, off = orc.cell_structures(g, w.pos, w.type)
    assert np.array_equal(np.sort(perm), np.arange(w.n, dtype=np.uint32))
    assert np.all(np.diff(ks.astype(np.int64)) >= 0)
    assert np.array_equal(ks, key[perm])
    same = ks[1:] == ks[:-1]
    assert same.sum() > 100
    assert np.all(perm[1:][same] > perm[:-1][same])          # ties keep slot order
    # equals numpy's stable argsort (library routine re-derivation)
    assert np.array_equal(perm, np.argsort(key, kind="stable").astype(np.uint32))


def test_cell_offsets(orc, c2small):
    w = c2small
    p = orc.params_from_workload(w)
    g = orc.grid_spec(p, [2, 2])
    key, ks, perm, off = orc.cell_structures(g, w.pos, w.type)
    ncell = g.base[g.n_types]
    assert off[0] == 0 and off[ncell] == w.n and len(off) == ncell + 1
    assert np.all(np.diff(off.astype(np.int64)) >= 0)
    assert np.array_equal(np.diff(off.astype(np.int64)), np.bincount(key, minlength=ncell))
    for c in np.unique(ks)[:50]:
        assert np.all(ks[off[c]:off[c + 1]] == c)


def test_clamp_and_nan(orc, c2small):
    w = c2small
    p = orc.params_from_workload(w)
    g = orc.grid_spec(p)
    x = np.array([[1e6, -1e6, 0.0], [np.nan, np.inf, -np.inf]], dtype=np.float32)
    key = orc.cell_structures(g, x, np.array([0, 0], np.int32))[0]
    G = g.G[0]
    assert key[0] == ((G // 2) * G + 0) * G + (G - 1)
    assert key[1] == (0 * G + (G - 1)) * G + 0


# ---- input generators ------------------------------------------------------

def test_type_counts():
    assert type_counts(32768, [0.7, 0.3]) == [22938, 9830]
    assert type_counts(250000, [0.5, 0.3, 0.2]) == [125000, 75000, 50000]
    assert sum(type_counts(1001, [0.5, 0.3, 0.2])) == 1001


@pytest.mark.parametrize("name,n", [("C1", None), ("C2", 4096), ("C3", 6000), ("C5", 5000)])
def test_ball_workloads(name, n):
    from scipy.spatial import cKDTree
    w = make_workload(name, n)
    assert w.pos.dtype == np.float32 and w.pos.shape == (w.n, 3)
    assert w.vel.dtype == np.float32 and w.type.dtype == np.int32
    assert np.array_equal(w.type, np.sort(w.type))            # ids blockwise by type
    assert list(np.bincount(w.type)) == type_counts(w.n, w.fractions)
    sig = np.asarray(w.sigma)[w.type]
    r = np.linalg.norm(w.pos.astype(np.float64), axis=1)
    assert np.all(r <= w.R0 - 0.5 * sig + 1e-4)
    pairs = cKDTree(w.pos.astype(np.float64)).query_pairs(0.9 * max(w.sigma), output_type="ndarray")
    if pairs.size:
        d = np.linalg.norm(w.pos[pairs[:, 0]].astype(np.float64) - w.pos[pairs[:, 1]], axis=1)
        assert np.all(d >= 0.9 * 0.5 * (sig[pairs[:, 0]] + sig[pairs[:, 1]]) - 1e-4)
    # uniform in the ball: <r^3>/R^3 = 1/2
    m = w.type == 0
    assert np.mean((r[m] / (w.R0 - 0.5 * w.sigma[0])) ** 3) == pytest.approx(0.5, abs=5 / np.sqrt(m.sum()))
    # Maxwell-Boltzmann: variance kT/m_a per component
    for a in range(w.n_types):
        v = w.vel[w.type == a]
        assert v.var() == pytest.approx(w.kT / w.mass[a], rel=6 * np.sqrt(2.0 / v.size))
    w2 = make_workload(name, n)
    assert np.array_equal(w.pos, w2.pos) and np.array_equal(w.vel, w2.vel)


def test_fcc_workload():
    from scipy.spatial import cKDTree
    w = make_workload("C4", n=8000)
    r = np.linalg.norm(w.pos.astype(np.float64), axis=1)
    assert w.n == 8000 and np.all(r <= w.R0 - 0.5 + 0.05 * np.sqrt(3) + 1e-4)
    phi = w.n * 0.125 / w.R0 ** 3
    assert phi == pytest.approx(0.40, rel=1e-12)
    d, _ = cKDTree(w.pos.astype(np.float64)).query(w.pos.astype(np.float64), k=2)
    assert d[:, 1].min() > 0.9 and np.median(d[:, 1]) == pytest.approx(1.2, abs=0.1)
    full = make_workload("C4", state=False)
    assert full.R0 == pytest.approx(42.749, abs=1e-3)
