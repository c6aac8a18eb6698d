"""Pins of oracle/observables.py (Eq. 2-4, 6, 8 of the paper and the cluster reading R23)
against closed forms, special cases and an independent library routine."""
import numpy as np
import pytest

from oracle import observables as O


def ball_points(rng, n, R):
    v = rng.normal(size=(n, 3))
    v /= np.linalg.norm(v, axis=1)[:, None]
    return v * (R * rng.random(n) ** (1.0 / 3.0))[:, None]


def fcc_ball(a, R):
    """All FCC sites (lattice constant a) inside the ball of radius R."""
    m = int(np.ceil(R / a)) + 1
    g = np.arange(-m, m + 1)
    c = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 3).astype(np.float64)
    basis = np.array([[0, 0, 0], [0.5, 0.5, 0], [0.5, 0, 0.5], [0, 0.5, 0.5]])
    x = (c[:, None, :] + basis[None, :, :]).reshape(-1, 3) * a
    return x[(x * x).sum(axis=1) <= R * R]


def test_rdf_of_an_ideal_gas_in_a_ball():
    """Eq. 6 as printed has no boundary correction: for uniform points in
    a ball of radius R it must return the ball pair-distance law
    g(r) = 1 - 3r/(4R) + r^3/(16 R^3)."""
    rng = np.random.default_rng(11)
    R, n = 10.0, 4000
    acc = []
    for _ in range(3):
        r, g = O.rdf(ball_points(rng, n, R), R, dr=0.25, r_max=8.0)
        acc.append(g)
    g = np.mean(acc, axis=0)
    exact = 1.0 - 3.0 * r / (4.0 * R) + r ** 3 / (16.0 * R ** 3)
    # pairs per bin ~ n^2/2 * 3 r^2 dr / R^3: > 1e4 beyond r = 1 -> < 1 % noise on the mean of 3
    sel = r > 1.0
    assert np.max(np.abs(g[sel] / exact[sel] - 1.0)) < 0.03
    assert abs(np.mean(g[sel] / exact[sel]) - 1.0) < 0.008      # sample-to-sample scatter ~ 0.3 %


def test_rdf_counts_ordered_pairs_once_each():
    """Two NPs at distance 1 in a sample of volume V: psi_1 = psi_2 = 1 in that shell, so
    g = (2/N) / ((N-1) dV/V) with N = 2."""
    R = 3.0
    x = np.array([[0.0, 0, 0], [1.02, 0, 0]])
    r, g = O.rdf(x, R, dr=0.1, r_max=2.0)
    k = 10                                    # shell [1.0, 1.1)
    V = 4.0 / 3.0 * np.pi * R ** 3
    dV = 4.0 / 3.0 * np.pi * (1.1 ** 3 - 1.0 ** 3)
    assert g[k] == pytest.approx((2.0 / 2.0) / (1.0 * dV / V), rel=1e-12)
    assert np.count_nonzero(g) == 1


def test_radial_concentration_uniform_and_normalised():
    """Eq. 8: uniform filling gives C = 1 in every shell; sum_k C_k dV_k / V = 1 always."""
    rng = np.random.default_rng(5)
    R = 7.0
    x = ball_points(rng, 200000, R)
    r, C = O.radial_concentration(x, R, dr=0.5)
    assert np.max(np.abs(C[3:] - 1.0)) < 0.05          # >= 2600 NPs per shell from k = 3
    edges = 0.5 * np.arange(len(C) + 1)
    V = 4.0 / 3.0 * np.pi * R ** 3
    assert np.sum(C * O.shell_volumes(edges) / V) == pytest.approx(1.0, rel=1e-12)
    # a thin surface layer: all weight in the last shell
    s = x / np.linalg.norm(x, axis=1)[:, None] * (R - 0.1)
    _, Cs = O.radial_concentration(s, R, dr=0.5)
    assert np.count_nonzero(Cs) == 1 and Cs[-1] > 1.0


def test_radius_of_gyration_closed_forms():
    # straight chain of N touching spheres of diameter d: R_g^2 = (N^2 - 1) d^2 / 12
    N, d = 101, 0.7
    x = np.zeros((N, 3))
    x[:, 0] = d * np.arange(N)
    assert O.radius_of_gyration(x) == pytest.approx(np.sqrt((N * N - 1) * d * d / 12.0), rel=1e-12)
    # translation invariance (Eq. 4 subtracts the centre of mass)
    assert O.radius_of_gyration(x + 123.0) == pytest.approx(O.radius_of_gyration(x), rel=1e-10)
    # two points at +-a: R_g = a
    assert O.radius_of_gyration(np.array([[-2.0, 0, 0], [2.0, 0, 0]])) == pytest.approx(2.0)


def test_fractal_dimension_of_compact_and_linear_aggregates():
    """k_f = 1.593 is the prefactor of a compact hexagonal structure: a
    close-packed ball of touching spheres must give D_f -> 3; a straight chain -> 1."""
    d = 1.0
    x = fcc_ball(a=np.sqrt(2.0) * d, R=14.0)          # nearest-neighbour distance = d
    assert len(x) > 15000
    assert O.fractal_dimension(x, d) == pytest.approx(3.0, abs=0.02)
    # chain: D_f = ln(N/k_f) / ln(2 R_g / d) with the closed-form R_g
    N = 4001
    c = np.zeros((N, 3))
    c[:, 2] = d * np.arange(N)
    exact = np.log(N / 1.593) / np.log(2.0 * np.sqrt((N * N - 1) / 12.0))
    assert O.fractal_dimension(c, d) == pytest.approx(exact, rel=1e-12)
    assert 1.0 < exact < 1.1
    # doubling every length leaves D_f unchanged if d_NP doubles too (Eq. 2 is a ratio)
    assert O.fractal_dimension(2.0 * x, 2.0 * d) == pytest.approx(O.fractal_dimension(x, d), rel=1e-12)


def test_clusters_hand_built():
    # a trimer (chain: 0-1, 1-2 bonded, 0-2 not), a dimer, a monomer
    x = np.array([[0, 0, 0], [1.2, 0, 0], [2.4, 0, 0], [10, 0, 0], [10, 1.4, 0], [20, 20, 20]], float)
    t = np.zeros(6, dtype=np.int32)
    lab = O.cluster_labels(x, t, [1.0], bond_factor=1.5)
    assert lab.tolist() == [0, 0, 0, 1, 1, 2]
    st = O.cluster_statistics(lab)
    assert st["n_clusters"] == 3 and st["largest"] == 3 and st["mean_size"] == 2.0
    assert st["log2_hist"].tolist() == [1, 2]           # sizes 1 | 2, 3
    # the bond length scales with sigma_ab: the same dimer of two large NPs, and mixed
    y = np.array([[0, 0, 0], [2.0, 0, 0]], float)
    assert O.cluster_labels(y, [0, 0], [1.0, 2.0]).tolist() == [0, 1]      # 2.0 >= 1.5
    assert O.cluster_labels(y, [1, 1], [1.0, 2.0]).tolist() == [0, 0]      # 2.0 < 3.0
    assert O.cluster_labels(y, [0, 1], [1.0, 2.0]).tolist() == [0, 0]      # 2.0 < 2.25


def test_clusters_equal_library_connected_components():
    sp = pytest.importorskip("scipy.sparse")
    from scipy.sparse.csgraph import connected_components
    rng = np.random.default_rng(3)
    n = 600
    x = rng.random((n, 3)) * 22.0            # ~1.4 bonds per NP: below percolation
    t = rng.integers(0, 2, n).astype(np.int32)
    sigma = np.array([1.0, 1.4])
    lab = O.cluster_labels(x, t, sigma, bond_factor=1.5)
    d = np.sqrt(((x[:, None, :] - x[None, :, :]) ** 2).sum(axis=2))
    lim = 1.5 * 0.5 * (sigma[t][:, None] + sigma[t][None, :])
    adj = (d < lim) & ~np.eye(n, dtype=bool)
    ncomp, ref = connected_components(sp.csr_matrix(adj), directed=False)
    assert lab.max() + 1 == ncomp and 5 < ncomp < n
    # same partition: the map label -> ref label is a bijection
    pairs = set(zip(lab.tolist(), ref.tolist()))
    assert len(pairs) == ncomp


def test_contract_histograms_equal_the_fp64_definitions():
    """oracle.rdf_hist / radial_hist (fp32 contract #4, the integers the CUDA path must
    reproduce bit for bit) against observables.rdf / radial_concentration (fp64,
    np.histogram, pinned above): the same counts except for distances that round
    across a bin edge, and exactly the same total."""
    import oracle
    from paper_2501_04456_b200 import workloads as W
    w = W.make_workload("C2", 3000)
    x = w.pos
    dr, nb = 0.25, 40
    h = oracle.rdf_hist(x, dr, nb)
    r, g = O.rdf(x.astype(np.float64), w.R0, dr, dr * nb)
    g2 = oracle.rdf_from_hist(h, w.n, w.R0, dr)
    # recover the fp64 counts from g and compare bin by bin
    V = 4.0 / 3.0 * np.pi * w.R0 ** 3
    edges = dr * np.arange(nb + 1)
    cnt64 = np.rint(g * w.n * (w.n - 1) * O.shell_volumes(edges) / V).astype(np.int64)
    assert h.sum() > 1e5 and h.sum() % 2 == 0                  # ordered pairs come in twos
    assert abs(int(h.sum()) - int(cnt64.sum())) <= 4
    assert np.max(np.abs(h.astype(np.int64) - cnt64)) <= 4     # only edge-rounding moves a pair
    assert np.allclose(g2[4:], g[4:], rtol=2e-3, atol=0)
    # radial profile, sums and N_surf
    ra = 0.5 * np.asarray(w.sigma)
    hr, sums, ns = oracle.radial_hist(x, w.type, ra, w.R0, 2.0, 30)
    x64 = x.astype(np.float64)
    rr = np.sqrt((x64 * x64).sum(axis=1))
    ref = np.histogram(rr, bins=2.0 * np.arange(31))[0]
    assert hr.sum() == w.n and np.max(np.abs(hr.astype(np.int64) - ref)) <= 2
    assert np.allclose(sums[:3], x64.sum(axis=0), rtol=0, atol=1e-9)
    assert sums[3] == pytest.approx((rr * rr).sum(), rel=1e-13)
    assert ns == int(np.count_nonzero(rr > w.R0 - 2.0 * ra[w.type]))
    # R_g from the sums (Eq. 3-4): <|x|^2> - |r_0|^2
    rg = np.sqrt(sums[3] / w.n - ((sums[:3] / w.n) ** 2).sum())
    assert rg == pytest.approx(O.radius_of_gyration(x64), rel=1e-12)


def test_contract_cluster_labels_equal_the_fp64_definition():
    """oracle.cluster_labels (fp32 bond predicate, min-label propagation in C) gives the
    same partition as observables.cluster_labels (fp64, union-find), which is pinned to
    scipy above."""
    import oracle
    from paper_2501_04456_b200 import workloads as W
    w = W.make_workload("C2", 3000)
    x = (w.pos * np.float32(0.6)).astype(np.float32)           # compress: plenty of bonds
    sg = np.asarray(w.sigma)
    sab = 0.5 * (sg[:, None] + sg[None, :])
    lab = oracle.cluster_labels(x, w.type, sab, 1.5)
    ref = O.cluster_labels(x.astype(np.float64), w.type, sg, 1.5)
    assert 10 < ref.max() + 1 < w.n
    pairs = set(zip(lab.tolist(), ref.tolist()))
    assert len(pairs) == ref.max() + 1 == len(set(lab.tolist()))
    # canonical: the label is the smallest member
    for l in np.unique(lab)[:50]:
        assert np.nonzero(lab == l)[0].min() == l
