"""Headless view (lv_render) against the oracle's restatement of the
same splat: every pixel bit-exact."""
import numpy as np
import pytest

from paper_2501_04456_b200 import tuning, workloads as W

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


@pytest.mark.parametrize("name,n,cpc,steps,WH,min_marks", [
    ("P1", None, None, 300, (720, 360), 30),          # Fig. 2's own scenario: isotropic centrifugal force, shell at the wall
    ("C3", 20000, [1, 2, 2], 200, (333, 171), 30),    # three sizes, moving interface, ragged map
    ("C4", 19999, [2], 3000, (512, 256), 0),          # dense lattice relaxing towards the wall
    ("C1", None, None, 0, (97, 64), 0),
])
def test_surface_map_bit_exact(B, orc, name, n, cpc, steps, WH, min_marks):
    """lv_render_surface (Fig. 2 left panel) against the oracle's per-pixel brute force."""
    w = W.make_workload(name, n)
    ra = 0.5 * np.asarray(w.sigma)
    sim = B.Simulation.from_workload(w, cells_per_cut=cpc if cpc is not None else tuning.cells_per_cut(w))
    if steps:
        sim.step(steps)
    x, v, t, R, st = sim.get_state()
    img = sim.render_surface(WH[0], WH[1], PAL, DROP)
    ref = orc.render_surface(x, t, ra, R, WH[0], WH[1], PAL, DROP)
    assert img.shape == ref.shape == (WH[1], WH[0])
    assert (ref != DROP).sum() >= min_marks
    assert np.array_equal(img, ref), int((img != ref).sum())
    dev = sim.render_surface(WH[0], WH[1], PAL, DROP, on_device=True)
    sim.synchronize()
    assert np.array_equal(dev.cpu().numpy().view(np.uint32), ref)
    # the map does not disturb the run
    ref_sim = B.Simulation.from_workload(w, cells_per_cut=cpc if cpc is not None else tuning.cells_per_cut(w))
    ref_sim.step(steps + 20); sim.step(20)
    xa, va, _, _, _ = sim.get_state()
    xb, vb, _, _, _ = ref_sim.get_state()
    assert np.array_equal(xa, xb) and np.array_equal(va, vb)
    sim.close(); ref_sim.close()


def test_surface_map_special_positions(B, orc):
    """NPs placed by hand: on the poles, on the date line, at the centre, outside, and one
    larger than the droplet -- the window logic of the kernel against the brute force."""
    w = W.make_workload("C2", 64)
    R = float(w.R0)
    x = np.zeros((64, 3), np.float32)
    rng = np.random.default_rng(3)
    d = rng.normal(size=(64, 3)); d /= np.linalg.norm(d, axis=1)[:, None]
    x[:] = (d * (R - 0.3)).astype(np.float32)
    x[0] = (0, 0, R); x[1] = (0, 0, -R + 0.2); x[2] = (-R, 0, 0); x[3] = (-R + 0.1, 1e-4, 0.3)
    x[4] = (0, 0, 0); x[5] = (R + 5, 0, 0); x[6] = (1e-9, 0, R - 0.4); x[7] = (0, R, 1e-3)
    x[8] = (R * 0.6, R * 0.8, 0); x[9] = (0.3, -0.2, R - 0.6)
    t = np.asarray(w.type[:64]).copy()
    ra = 0.5 * np.asarray(w.sigma)
    sim = B.Simulation.from_workload(w, load_state=False)
    sim.set_state(x, np.zeros_like(x), t, 0)
    for WH in ((360, 180), (64, 32), (1, 1), (1000, 7)):
        img = sim.render_surface(WH[0], WH[1], PAL, DROP)
        ref = orc.render_surface(x, t, ra, R, WH[0], WH[1], PAL, DROP)
        assert np.array_equal(img, ref), (WH, int((img != ref).sum()))
    with pytest.raises(B.LvError):
        sim.render_surface(0, 10, PAL)
    with pytest.raises(B.LvError):
        sim.render_surface(10, 9000, PAL)
    sim.close()


def test_argument_checks(B):
    w = W.make_workload("C1")
    sim = B.Simulation.from_workload(w)
    for bad in (dict(eye=0.0), dict(f=-1.0), dict(W=0), dict(H=9000)):
        kw = dict(eye=70.0, f=900.0, W=64, H=64)
        kw.update(bad)
        with pytest.raises(B.LvError):
            sim.render(kw["eye"], kw["f"], 0.0, 0.0, kw["W"], kw["H"], PAL)
    sim.close()
