"""Headless view (lv_render) against the oracle's restatement of the
same splat: every pixel bit-exact."""
import numpy as np
import pytest

from paper_2501_04456_b200 import workloads as W

pytestmark = pytest.mark.gpu

PAL = [0x00ff8040, 0x004080ff, 0x0040ff80]
BG, DROP = 0xff000000, 0xff201008


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


@pytest.mark.parametrize("name,n,cpc,view", [
    ("C1", None, None, dict(eye=70.0, f=900.0, yaw=0.3, pitch=-0.2, W=640, H=480)),
    ("C3", 20000, [1, 2, 2], dict(eye=260.0, f=700.0, yaw=1.1, pitch=0.7, W=333, H=257)),   # ragged
    ("C4", 19999, [2], dict(eye=30.0, f=300.0, yaw=0.0, pitch=0.0, W=256, H=256)),          # camera close: clipping
    ("C2", 8191, [2, 2], dict(eye=25.0, f=200.0, yaw=2.0, pitch=1.3, W=128, H=96)),         # camera INSIDE the droplet
])
def test_image_bit_exact(B, orc, name, n, cpc, view):
    w = W.make_workload(name, n)
    ra = 0.5 * np.asarray(w.sigma)
    sim = B.Simulation.from_workload(w, cells_per_cut=cpc)
    for steps in (0, 40):
        if steps:
            sim.step(steps)
        x, v, t, R, st = sim.get_state()
        img = sim.render(view["eye"], view["f"], view["yaw"], view["pitch"], view["W"], view["H"], PAL,
                         BG, DROP)
        ref = orc.render(x, t, ra, R, view["eye"], view["f"], view["yaw"], view["pitch"], view["W"],
                         view["H"], PAL, BG, DROP)
        assert img.shape == ref.shape == (view["H"], view["W"])
        drawn = (ref != BG) & (ref != DROP)
        assert drawn.sum() > 50
        assert np.array_equal(img, ref), int((img != ref).sum())
        dev = sim.render(view["eye"], view["f"], view["yaw"], view["pitch"], view["W"], view["H"], PAL,
                         BG, DROP, on_device=True)
        sim.synchronize()
        assert np.array_equal(dev.cpu().numpy().view(np.uint32), ref)
    # the view does not disturb the run
    ref_sim = B.Simulation.from_workload(w, cells_per_cut=cpc)
    ref_sim.step(80); sim.step(40)
    xa, va, _, _, _ = sim.get_state()
    xb, vb, _, _, _ = ref_sim.get_state()
    assert np.array_equal(xa, xb) and np.array_equal(va, vb)
    sim.close(); ref_sim.close()


def test_argument_checks(B):
    w = W.make_workload("C1")
    sim = B.Simulation.from_workload(w)
    for bad in (dict(eye=0.0), dict(f=-1.0), dict(W=0), dict(H=9000)):
        kw = dict(eye=70.0, f=900.0, W=64, H=64)
        kw.update(bad)
        with pytest.raises(B.LvError):
            sim.render(kw["eye"], kw["f"], 0.0, 0.0, kw["W"], kw["H"], PAL)
    sim.close()
