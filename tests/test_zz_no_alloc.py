"""lv_observe_rdf_noalloc: the RDF pair walk with its histogram scratch in a static device array
of the library (no cudaMalloc, no caller scratch).  Collected last on purpose (the suite runs with
pytest -x).  The result must equal the existing path's (lv_observe_rdf): the histogram is
integer work decided by fp32 contract #4 -> bit-exact, g(r) the same normalisation -> equal to
rounding; on two calls in a row (the array keeps the previous call's counts and must be
cleared), with different bin counts and on different handles, and sizes beyond the maximum are
rejected with LV_E_CAPACITY.  Passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

from paper_2501_04456_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2501_04456_b200 import binding
    binding.load()
    return binding


def same(B, sim, dr, nb):
    h0, g0 = sim.observe_rdf(dr, nb)
    h1, g1 = sim.observe_rdf_noalloc(dr, nb)
    assert h0.sum() > 0
    assert np.array_equal(h1, h0)                       # bit-exact
    assert np.allclose(g1, g0, rtol=1e-15, atol=0.0)
    return h0


def test_noalloc_rdf_equals_the_existing_path_twice_in_a_row(B):
    w = W.make_workload("C3", 20000)
    sim = B.Simulation.from_workload(w, cells_per_cut=[1, 2, 2])
    a = same(B, sim, 0.25, 33)                          # first call on this device: takes the symbol address
    b = same(B, sim, 0.25, 33)                          # second call: the array holds the first call's counts
    assert np.array_equal(a, b)
    c = same(B, sim, 0.05, 150)                         # more bins than before ...
    d = same(B, sim, 0.5, 7)                            # ... and fewer: stale counts beyond n_bins never read
    assert c.sum() != d.sum()
    sim.step(25)                                        # a moved state, moving interface
    same(B, sim, 0.25, 33)
    # another handle shares the same array
    w2 = W.make_workload("C1")
    sim2 = B.Simulation.from_workload(w2)
    same(B, sim2, 0.05, 100)
    same(B, sim, 0.25, 33)
    # the calls leave the run bit-identical
    ref = B.Simulation.from_workload(w, cells_per_cut=[1, 2, 2])
    ref.step(35)
    sim.step(10)
    for u, v in zip(sim.get_state()[:3], ref.get_state()[:3]):
        assert np.array_equal(u, v)
    for s in (sim, sim2, ref):
        s.close()


def test_noalloc_rdf_at_the_maximum_and_beyond(B):
    w = W.make_workload("C1")
    sim = B.Simulation.from_workload(w)
    same(B, sim, 0.001, B.NOALLOC_MAX_BINS)             # the whole array
    with pytest.raises(B.LvError) as e:
        sim.observe_rdf_noalloc(0.001, B.NOALLOC_MAX_BINS + 1)
    assert e.value.code == B.E_CAPACITY
    same(B, sim, 0.05, 100)                             # still usable after the rejected call
    sim.close()
