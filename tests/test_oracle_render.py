"""Pins of the oracle's headless view (oracle.render): the splat is
this build's own definition of Fig. 2's perspective panel (include/lv.h: lv_view), so it is
pinned to projective geometry -- disc areas, positions, occlusion, orientation, shading."""
import numpy as np

import oracle

PAL = [0x00ff8040, 0x004080ff]
BG, DROP = 0xff000000, 0xff201008


def img(x, t, ra, R=20.0, eye=100.0, f=400.0, yaw=0.0, pitch=0.0, W=201, H=161):
    return oracle.render(np.asarray(x, np.float32), np.asarray(t, np.int32), ra, R, eye, f, yaw, pitch,
                         W, H, PAL, BG, DROP)


def test_single_sphere_disc_area_centre_and_shading():
    im = img([[0, 0, 0]], [0], [2.0])
    cov = (im != BG) & (im != DROP)
    rho = 400.0 * 2.0 / 100.0                      # f r / zc = 8 px
    assert abs(cov.sum() - np.pi * rho * rho) < 0.06 * np.pi * rho * rho
    ys, xs = np.nonzero(cov)
    assert abs(xs.mean() - 100.0) < 0.51 and abs(ys.mean() - 80.0) < 0.51      # image centre
    # brightest at the centre (normal towards the camera): palette * (0.25 + 0.75 nz), nz ~ 1
    c = int(im[80, 100])
    assert (c >> 24) == 0xff
    assert abs((c & 0xff) - 0x40) <= 1 and abs(((c >> 8) & 0xff) - 0x80) <= 1 and abs(((c >> 16) & 0xff) - 0xff) <= 1
    # limb darkening: the rim is at ~ 0.25 of the base colour
    rim = int(im[80, 100 + 7])
    assert ((rim >> 16) & 0xff) < ((c >> 16) & 0xff)
    # droplet silhouette: disc of radius f R / eye = 80 px, clipped by the 201 x 161 frame
    sil = im == DROP
    yy, xx = np.mgrid[0:161, 0:201]
    inside = ((xx + 0.5 - 100.5) ** 2 + (yy + 0.5 - 80.5) ** 2) <= 80.0 ** 2
    assert np.array_equal(sil | cov, inside)


def test_perspective_scale_position_and_occlusion():
    # x to the right, y up; nearer spheres are larger
    im = img([[10, 0, 0], [0, 5, 0]], [0, 1], [1.0, 1.0])
    a = (im & 0xffffff) != 0
    ys, xs = np.nonzero((im != BG) & (im != DROP))
    assert xs.max() > 100 + 35 and ys.min() < 80 - 15            # +x -> right (40 px), +y -> up (20 px)
    near = img([[0, 0, 50]], [0], [1.0])
    far = img([[0, 0, -50]], [0], [1.0])
    n_near = ((near != BG) & (near != DROP)).sum()
    n_far = ((far != BG) & (far != DROP)).sum()
    assert n_near / n_far == np.float64(n_near) / n_far and 7.0 < n_near / n_far < 11.0   # (150/50)^2 = 9
    # occlusion: the sphere nearer to the camera (type 1, z = +5) hides the one behind it
    both = img([[0, 0, -5], [0, 0, 5]], [0, 1], [1.0, 1.0])
    c = int(both[80, 100])
    assert abs((c & 0xff) - 0xff) <= 1 and abs(((c >> 16) & 0xff) - 0x40) <= 1     # palette[1]
    # ... independent of the order of the NPs
    swapped = img([[0, 0, 5], [0, 0, -5]], [1, 0], [1.0, 1.0])
    assert np.array_equal(both, swapped)
    # behind the camera: nothing drawn
    none = img([[0, 0, 150]], [0], [1.0])
    assert not ((none != BG) & (none != DROP)).any()


def test_rotation_orientation():
    # yaw = +90 deg about y brings +x onto ... the view axis: x' = cy x + sy z, z' = -sy x + cy z
    r = oracle.view_rotation(np.pi / 2, 0.0).reshape(3, 3).astype(np.float64)
    assert np.allclose(r @ np.array([0, 0, 1.0]), [1, 0, 0], atol=1e-6)      # +z appears on the right
    assert np.allclose(r @ r.T, np.eye(3), atol=1e-6) and np.linalg.det(r) > 0.999
    p = oracle.view_rotation(0.0, np.pi / 2).reshape(3, 3).astype(np.float64)
    assert np.allclose(p @ np.array([0, 1.0, 0]), [0, 0, 1], atol=1e-6)      # pitch tips +y towards the camera
    im0 = img([[0, 0, 10]], [0], [1.0])
    im1 = img([[0, 0, 10]], [0], [1.0], yaw=np.pi / 2)
    x0 = np.nonzero((im0 != BG) & (im0 != DROP))[1].mean()
    x1 = np.nonzero((im1 != BG) & (im1 != DROP))[1].mean()
    assert abs(x0 - 100.0) < 0.6 and abs(x1 - (100.5 + 40.0 - 0.5)) < 0.6


def test_per_np_splat_equals_the_per_pixel_definition():
    """lvo_render walks, per NP, the bounding box of its projected disc (the structure the CUDA
    splat mirrors); lvo_render_pixels is the definition -- every pixel against every NP, no
    boxes.  Bit-identical images on crowded, clipped, close-up and inside-the-droplet scenes pin
    the bounding-box logic to something that does not share it."""
    rng = np.random.default_rng(7)
    pal = [0x00ff8040, 0x004080ff, 0x0040ff80]
    for n, R, eye, focal, yaw, pitch, W, H in (
            (400, 10.0, 30.0, 120.0, 0.3, -0.2, 96, 64),        # the whole droplet
            (400, 10.0, 12.0, 200.0, 1.1, 0.4, 77, 53),         # close: discs clipped by the frame
            (300, 10.0, 4.0, 60.0, -0.7, 0.9, 64, 48),          # camera INSIDE: NPs behind / around it
            (50, 3.0, 500.0, 40.0, 0.0, 0.0, 33, 31),           # far: sub-pixel discs
            (0, 5.0, 20.0, 50.0, 0.0, 0.0, 16, 9)):             # empty
        x = rng.normal(0, 1, size=(n, 3))
        x *= (R * rng.random(n) ** (1 / 3) / np.maximum(np.linalg.norm(x, axis=1), 1e-9))[:, None]
        t = rng.integers(0, 3, size=n).astype(np.int32)
        ra = [0.4, 0.7, 1.3]
        a = oracle.render(x.astype(np.float32), t, ra, R, eye, focal, yaw, pitch, W, H, pal, BG, DROP)
        b = oracle.render(x.astype(np.float32), t, ra, R, eye, focal, yaw, pitch, W, H, pal, BG, DROP,
                          per_pixel=True)
        assert np.array_equal(a, b)
        if n:
            assert ((a != BG) & (a != DROP)).any()
