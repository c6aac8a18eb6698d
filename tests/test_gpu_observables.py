"""On-device observables (lv_observe_rdf / lv_observe_radial) against
the oracle: the histograms are integers decided by fp32 contract #4 and must be bit-exact;
the fp64 sums (centre, R_g, D_f) agree to rounding; g(r) and the concentration profile are
the normalisations of Eq. 6 / Eq. 8."""
import numpy as np
import pytest

from paper_2501_04456_b200 import workloads as W

pytestmark = pytest.mark.gpu


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


CASES = [  # (config, n, cells_per_cut, dr, n_bins of the RDF)
    ("C1", None, None, 0.05, 100),          # r <= 5 sigma = 2 r_c: wider than the force stencil
    ("C2", 8191, [2, 2], 0.1, 64),
    ("C3", 20000, [1, 2, 2], 0.25, 33),     # ragged: r_max = 8.25
    ("C4", 19999, [2], 0.02, 150),
]


@pytest.mark.parametrize("name,n,cpc,dr,nb", CASES)
def test_rdf_histogram_bit_exact_and_normalised(B, orc, name, n, cpc, dr, nb):
    from oracle import observables as O
    w = W.make_workload(name, n)
    sim = B.Simulation.from_workload(w, cells_per_cut=cpc)
    h, g = sim.observe_rdf(dr, nb)
    ho = orc.rdf_hist(w.pos, dr, nb)
    assert ho.sum() > 0
    assert np.array_equal(h, ho)                                    # integers: bit-exact
    assert np.allclose(g, orc.rdf_from_hist(ho, w.n, w.R0, dr), rtol=1e-13, atol=0)
    # ... and Eq. 6 written out in fp64 (np.histogram) agrees up to edge rounding
    _, g64 = O.rdf(w.pos.astype(np.float64), w.R0, dr, dr * nb)
    big = ho > 2000
    if big.any():
        assert np.allclose(g[big], g64[big], rtol=5e-3, atol=0)
    # after some steps (moving interface for C2/C3: V uses R(step)), again bit-exact
    sim.step(25)
    x, v, t, R, st = sim.get_state()
    h2, g2 = sim.observe_rdf(dr, nb)
    ho2 = orc.rdf_hist(x, dr, nb)
    assert np.array_equal(h2, ho2)
    assert np.allclose(g2, orc.rdf_from_hist(ho2, w.n, R, dr), rtol=1e-13, atol=0)
    # the observable does not disturb the run
    ref = B.Simulation.from_workload(w, cells_per_cut=cpc)
    ref.step(50)
    sim.step(25)
    xa, va, _, _, _ = sim.get_state()
    xb, vb, _, _, _ = ref.get_state()
    assert np.array_equal(xa, xb) and np.array_equal(va, vb)
    sim.close(); ref.close()


@pytest.mark.parametrize("name,n,cpc,dr,nb", CASES)
def test_radial_profile_sums_and_surface_count(B, orc, name, n, cpc, dr, nb):
    from oracle import observables as O
    w = W.make_workload(name, n)
    sim = B.Simulation.from_workload(w, cells_per_cut=cpc)
    sim.step(10)
    x, v, t, R, st = sim.get_state()
    drr = R / 37.0                                                  # shells up to the interface
    out = sim.observe_radial(drr, 40)
    ra = 0.5 * np.asarray(w.sigma)
    ho, sums, ns = orc.radial_hist(x, w.type, ra, R, drr, 40)
    assert np.array_equal(out["hist"], ho) and ho.sum() == w.n
    assert out["n_surf"] == ns
    x64 = x.astype(np.float64)
    assert np.allclose(out["centre"], sums[:3] / w.n, rtol=0, atol=1e-11)
    assert out["r_g"] == pytest.approx(O.radius_of_gyration(x64), rel=1e-11)
    d_np = float(np.mean(np.asarray(w.sigma)[w.type]))
    assert out["d_f"] == pytest.approx(O.fractal_dimension(x64, d_np), rel=1e-10)
    # Eq. 8 from the oracle's counts
    k = np.arange(40)
    dV = 4.0 / 3.0 * np.pi * (((k + 1) * drr) ** 3 - (k * drr) ** 3)
    V = 4.0 / 3.0 * np.pi * R ** 3
    assert np.allclose(out["conc"], (ho / w.n) / (dV / V), rtol=1e-13, atol=0)
    sim.close()


def test_observables_with_the_neighbour_list_on(B, orc):
    """lv_observe_rdf rebuilds the cells; a skin-list run must not notice."""
    w = W.make_workload("C2", 8191)
    a = B.Simulation.from_workload(w, cells_per_cut=[2, 2], neighbour_list=(0.4, 256))
    b = B.Simulation.from_workload(w, cells_per_cut=[2, 2], neighbour_list=(0.4, 256))
    a.step(30); b.step(30)
    x, _, _, _, _ = a.get_state()
    h, _ = a.observe_rdf(0.1, 50)
    assert np.array_equal(h, orc.rdf_hist(x, 0.1, 50))
    a.observe_radial(1.0, 64)
    a.step(30); b.step(30)
    xa, va, _, _, _ = a.get_state()
    xb, vb, _, _, _ = b.get_state()
    assert np.array_equal(xa, xb) and np.array_equal(va, vb)
    a.close(); b.close()


def test_argument_checks(B):
    w = W.make_workload("C1")
    sim = B.Simulation.from_workload(w)
    for bad in ((0.0, 10), (0.1, 0), (0.1, 9000), (-1.0, 10)):
        with pytest.raises(B.LvError):
            sim.observe_rdf(*bad)
        with pytest.raises(B.LvError):
            sim.observe_radial(*bad)
    sim.close()


@pytest.mark.parametrize("name,n,cpc,scale,steps", [
    ("C1", None, None, 1.0, 0),
    ("C1", None, None, 1.0, 3000),            # the LJ gas has started to condense
    ("C2", 8191, [2, 2], 0.6, 0),             # compressed: large aggregates
    ("C3", 20000, [1, 2, 2], 0.5, 0),
    ("C4", 19999, [2], 1.0, 0),               # dense: one percolating aggregate + a few
])
def test_aggregates_equal_the_oracle_partition(B, orc, name, n, cpc, scale, steps):
    from oracle import observables as O
    w = W.make_workload(name, n)
    if scale != 1.0:
        w.pos = (w.pos * np.float32(scale)).astype(np.float32)
    sim = B.Simulation.from_workload(w, cells_per_cut=cpc)
    if steps:
        sim.step(steps)
    x, v, t, R, st = sim.get_state(check=False)
    out = sim.observe_clusters(1.5)
    sg = np.asarray(w.sigma)
    lab = orc.cluster_labels(x, w.type, 0.5 * (sg[:, None] + sg[None, :]), 1.5)
    assert np.array_equal(out["labels"], lab)                 # canonical labels: bit-exact
    stats = O.cluster_statistics(np.unique(lab, return_inverse=True)[1])
    assert out["n_clusters"] == stats["n_clusters"]
    assert out["largest"] == stats["largest"]
    assert out["mean_size"] == pytest.approx(stats["mean_size"], rel=1e-14)
    hist = np.zeros(32, dtype=np.uint64)
    hist[:len(stats["log2_hist"])] = stats["log2_hist"]
    assert np.array_equal(out["log2_hist"], hist)
    # statistics only (no label transfer) give the same numbers
    out2 = sim.observe_clusters(1.5, want_labels=False)
    assert out2["labels"] is None and out2["n_clusters"] == out["n_clusters"]
    # a bond longer than the cut-off cannot be searched in the force stencil
    with pytest.raises(B.LvError):
        sim.observe_clusters(100.0)
    sim.close()
