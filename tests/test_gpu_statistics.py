"""Long-run statistical parity (BASELINE north star; SURVEY sec. 8(c) "Long runs"):
trajectories are chaotic, so after thousands of steps the CUDA path and the fp64 oracle
are compared through the paper's own observables -- RDF (Eq. 6), aggregate statistics
(R23) and the fractal dimension (Eq. 2-4) -- averaged over time and over seeds.

Bounds: RDF first-peak bin equal +-1, peak height within 5 %,
int |dg| dr / int g dr <= 0.03; number of aggregates and mean aggregate size within
10 %; aggregate-size histogram (mass in log2 size classes) within total-variation
distance 0.05; D_f within +-0.02; each widened to 3 standard errors of the oracle's own
seed-to-seed scatter where that is larger."""
import numpy as np
import pytest

from paper_2501_04456_b200 import workloads as W

pytestmark = pytest.mark.gpu

DR, RMAX = 0.05, 5.0
NCLASS = 24


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


def observe(O, x, w, R):
    _, g = O.rdf(x, R, DR, RMAX)
    lab = O.cluster_labels(x, w.type, w.sigma)
    st = O.cluster_statistics(lab)
    # aggregate-size histogram, mass-weighted: fraction of the NPs that sit in aggregates of
    # size [2^k, 2^(k+1))
    sizes = np.bincount(lab)
    mass = np.bincount(np.floor(np.log2(sizes)).astype(np.int64), weights=sizes, minlength=NCLASS)
    return g, np.array([st["n_clusters"], st["mean_size"]], dtype=np.float64), \
        O.fractal_dimension(x, float(np.mean(np.asarray(w.sigma)[w.type]))), mass / len(lab)


def time_average(samples):
    g = np.mean([s[0] for s in samples], axis=0)
    cl = np.mean([s[1] for s in samples], axis=0)
    df = float(np.mean([s[2] for s in samples]))
    return g, cl, df, np.mean([s[3] for s in samples], axis=0)


def run_oracle(orc, O, w, n_steps, every, first):
    p = orc.params_from_workload(w)
    x, v = w.pos.astype(np.float64), w.vel.astype(np.float64)
    out = []
    for done in range(0, n_steps, every):
        x, v, bad = orc.step(p, x, v, w.type, step0=done, nsteps=every)
        assert bad == 0
        if done + every >= first:
            out.append(observe(O, x, w, orc.radius(p, done + every)))
    return time_average(out)


def run_gpu(B, orc, O, w, n_steps, every, first, cpc):
    p = orc.params_from_workload(w)
    sim = B.Simulation.from_workload(w, cells_per_cut=cpc)
    out = []
    for done in range(0, n_steps, every):
        sim.step(every)
        if done + every >= first:
            x, v, t, R, st = sim.get_state()
            assert st == done + every
            assert R == pytest.approx(orc.radius(p, done + every), rel=1e-12)
            out.append(observe(O, x.astype(np.float64), w, R))
    assert sim.status() == 0
    sim.close()
    return time_average(out)


def widened(bound, orc_values):
    """max(stated bound, 3 standard errors of the difference of two seed means)."""
    v = np.asarray(orc_values, dtype=np.float64)
    if len(v) < 2:
        return bound
    return max(bound, 3.0 * v.std(ddof=1) * np.sqrt(2.0 / len(v)))


@pytest.mark.parametrize("name,n,seeds,n_steps,every,cpc", [
    ("C1", None, (1, 2, 3), 8000, 250, None),        # LJ gas condensing in a fixed droplet
    ("C2", 4096, (2, 12), 3000, 250, [2, 2]),        # charged two-size mixture, shrinking droplet
    ("C4", 4096, (4, 14), 3000, 250, [3]),           # dense sticky LJ: late-stage aggregation
])
def test_long_run_statistics(B, orc, name, n, seeds, n_steps, every, cpc):
    from oracle import observables as O
    first = n_steps // 2
    go, gg, co, cg, do, dg, ho, hg = [], [], [], [], [], [], [], []
    for seed in seeds:
        w = W.make_workload(name, n, seed=seed)
        g, c, d, h = run_oracle(orc, O, w, n_steps, every, first)
        go.append(g); co.append(c); do.append(d); ho.append(h)
        g, c, d, h = run_gpu(B, orc, O, w, n_steps, every, first, cpc)
        gg.append(g); cg.append(c); dg.append(d); hg.append(h)
    go, gg, co, cg = np.array(go), np.array(gg), np.array(co), np.array(cg)
    g_o, g_g = go.mean(axis=0), gg.mean(axis=0)

    # RDF: position and height of the first peak, integrated difference
    ko, kg = int(np.argmax(g_o)), int(np.argmax(g_g))
    assert g_o[ko] > 1.5                                  # there is a contact peak to compare
    assert abs(ko - kg) <= 1
    tol_h = widened(0.05 * g_o[ko], go[:, ko])
    assert abs(g_g[ko] - g_o[ko]) <= tol_h, (g_g[ko], g_o[ko], tol_h)
    l1 = np.abs(g_g - g_o).sum() / g_o.sum()
    l1_seed = max(np.abs(go[i] - g_o).sum() / g_o.sum() for i in range(len(seeds)))
    assert l1 <= max(0.03, 3.0 * l1_seed * np.sqrt(2.0 / len(seeds))), (l1, l1_seed)

    # aggregates: number and mean size within 10 %
    for k, what in enumerate(("n_clusters", "mean_size")):
        tol = widened(0.10 * co[:, k].mean(), co[:, k])
        assert abs(cg[:, k].mean() - co[:, k].mean()) <= tol, (what, cg[:, k], co[:, k])

    # aggregate-size histogram (mass-weighted log2 classes): total-variation distance <= 0.05,
    # widened to 3 s.e. of the oracle's own seed-to-seed distance
    ho, hg = np.array(ho), np.array(hg)
    tv = 0.5 * np.abs(hg.mean(axis=0) - ho.mean(axis=0)).sum()
    tv_seed = max(0.5 * np.abs(ho[i] - ho.mean(axis=0)).sum() for i in range(len(seeds)))
    assert tv <= max(0.05, 3.0 * tv_seed * np.sqrt(2.0 / len(seeds))), (tv, tv_seed, ho, hg)
    print(f"\n{name}: size-class masses oracle {np.round(ho.mean(axis=0)[:12], 3)} GPU "
          f"{np.round(hg.mean(axis=0)[:12], 3)} TV {tv:.4f} (seed {tv_seed:.4f})")

    print(f"\n{name}: peak bin {ko}/{kg} height {g_o[ko]:.3f}/{g_g[ko]:.3f} L1 {l1:.4f} (seed {l1_seed:.4f}) "
          f"clusters {co[:, 0].mean():.1f}/{cg[:, 0].mean():.1f} mean size {co[:, 1].mean():.3f}/"
          f"{cg[:, 1].mean():.3f} D_f {np.mean(do):.4f}/{np.mean(dg):.4f}   (oracle/GPU)")
    # fractal dimension (Eq. 2 over all NPs of the droplet, as the paper does)
    assert abs(np.mean(dg) - np.mean(do)) <= widened(0.02, do), (dg, do)
