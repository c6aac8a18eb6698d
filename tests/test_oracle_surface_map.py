"""Pins of the oracle's surface map (oracle.render_surface; Fig. 2 left
panel).  The projection is this build's reading (equirectangular, include/lv.h),
so the oracle is pinned to spherical geometry: cap solid angles, the 1/cos(latitude)
elongation the caption describes, orientation, the date line, the poles, which NPs reach the
surface at all, and nearest-wins."""
import numpy as np

import oracle

PAL = [0x00ff8040, 0x004080ff]
DROP = 0xff201008
W, H = 720, 360
R = 20.0


def smap(x, t, ra, R=R, W=W, H=H):
    return oracle.render_surface(np.asarray(x, np.float32), np.asarray(t, np.int32), ra, R, W, H,
                                 PAL, DROP)


def solid_angle(mask):
    """sum of pixel solid angles cos(phi) dphi dlambda over the marked pixels"""
    Hh, Ww = mask.shape
    phi = np.pi / 2 - np.pi * (np.arange(Hh) + 0.5) / Hh
    return float((mask * np.cos(phi)[:, None]).sum() * (np.pi / Hh) * (2 * np.pi / Ww))


def cap_angle(d, r, R=R):
    """angular radius of the part of the sphere |s| = R inside the ball |s - x| < r, |x| = d"""
    return np.arccos((R * R + d * d - r * r) / (2 * R * d))


def at(lam_deg, phi_deg, d):
    lam, phi = np.radians(lam_deg), np.radians(phi_deg)
    return [d * np.cos(phi) * np.cos(lam), d * np.cos(phi) * np.sin(lam), d * np.sin(phi)]


def test_cap_solid_angle_on_inside_and_outside_the_surface():
    for d, r, k in ((R, 2.0, 1), (R - 1.0, 2.0, 1), (R + 1.5, 2.0, 1), (R - 0.4, 0.5, 4)):
        m = smap([at(30.0, 10.0, d)], [0], [r], W=k * W, H=k * H) != DROP
        want = 2 * np.pi * (1 - np.cos(cap_angle(d, r)))
        assert abs(solid_angle(m) - want) < 0.04 * want, (d, r)
    # colour and alpha
    im = smap([at(0.0, 0.0, R)], [1], [1.0, 2.0])
    assert set(np.unique(im)) == {DROP, 0xff000000 | PAL[1]}


def test_np_that_does_not_reach_the_surface_leaves_no_mark():
    assert (smap([at(10, 20, R - 2.01)], [0], [2.0]) == DROP).all()     # deeper than its radius
    assert (smap([at(10, 20, R + 2.01)], [0], [2.0]) == DROP).all()     # outside, not touching
    assert (smap([[0, 0, 0]], [0], [2.0]) == DROP).all()
    assert (smap([at(10, 20, R - 1.99)], [0], [2.0]) != DROP).any()


def test_elongation_with_latitude_as_in_the_caption():
    """'circles elongated due to the projection': the extent in longitude grows as
    asin(sin(alpha)/cos(phi)), the extent in latitude stays 2 alpha."""
    alpha = cap_angle(R, 2.0)
    for phi_deg in (0.0, 45.0, 60.0, 75.0):
        m = smap([at(0.0, phi_deg, R)], [0], [2.0]) != DROP
        ys, xs = np.nonzero(m)
        wid = (xs.max() - xs.min() + 1) * 360.0 / W
        hei = (ys.max() - ys.min() + 1) * 180.0 / H
        want_w = 2 * np.degrees(np.arcsin(np.sin(alpha) / np.cos(np.radians(phi_deg))))
        assert abs(wid - want_w) <= 1.01 and abs(hei - 2 * np.degrees(alpha)) <= 1.01, phi_deg


def test_orientation_longitude_latitude_and_date_line():
    def centre(lam, phi):
        m = smap([at(lam, phi, R)], [0], [1.5]) != DROP
        ys, xs = np.nonzero(m)
        return xs.mean(), ys.mean()
    cx, cy = centre(0.0, 0.0)                       # +x axis: middle of the map
    assert abs(cx - (W / 2 - 0.5)) < 0.6 and abs(cy - (H / 2 - 0.5)) < 0.6
    cx, cy = centre(90.0, 0.0)                      # +y axis: three quarters across
    assert abs(cx - (0.75 * W - 0.5)) < 0.6
    cx, cy = centre(-90.0, 30.0)                    # -y axis, northern latitude: upper left quarter
    assert abs(cx - (0.25 * W - 0.5)) < 0.6 and abs(cy - ((90 - 30) / 180 * H - 0.5)) < 0.6
    # -x axis: the mark is split between the left and the right edge of the map
    m = smap([at(180.0, 0.0, R)], [0], [1.5]) != DROP
    cols = np.nonzero(m.any(axis=0))[0]
    assert cols.min() == 0 and cols.max() == W - 1 and not m[:, W // 4: 3 * W // 4].any()
    assert abs(solid_angle(m) - 2 * np.pi * (1 - np.cos(cap_angle(R, 1.5)))) < 0.04 * solid_angle(m)


def test_pole_covers_whole_rows():
    alpha = cap_angle(R, 2.0)
    for z, rows in ((R, slice(0, None)), (-R, slice(None, None, -1))):
        m = (smap([[0.0, 0.0, z]], [0], [2.0]) != DROP)[rows]
        full = m.all(axis=1)
        n_rows = int(full.sum())
        assert full[:n_rows].all() and not m[n_rows:].any()          # full rows, then nothing
        assert abs(n_rows - np.degrees(alpha) / 180 * H) <= 1.0


def test_nearest_centre_wins_and_order_does_not_matter():
    a, b = at(0.0, 0.0, R), at(4.0, 0.0, R - 0.5)                     # overlapping marks, two types
    im = smap([a, b], [0, 1], [1.5, 1.5])
    assert np.array_equal(im, smap([b, a], [1, 0], [1.5, 1.5]))
    ys, xs = np.nonzero(im != DROP)
    # each marked pixel carries the colour of the NP whose centre is nearer to its surface point
    phi = np.pi / 2 - np.pi * (ys + 0.5) / H
    lam = -np.pi + 2 * np.pi * (xs + 0.5) / W
    s = R * np.stack([np.cos(phi) * np.cos(lam), np.cos(phi) * np.sin(lam), np.sin(phi)], axis=1)
    da = np.linalg.norm(s - np.array(a), axis=1)
    db = np.linalg.norm(s - np.array(b), axis=1)
    clear = np.abs(da - db) > 1e-4
    want = np.where(da < db, 0xff000000 | PAL[0], 0xff000000 | PAL[1])
    assert clear.sum() > 50 and np.array_equal(im[ys, xs][clear], want[clear])
    assert {int(v) for v in np.unique(im)} == {DROP, 0xff000000 | PAL[0], 0xff000000 | PAL[1]}


def test_shell_of_nps_covers_the_expected_fraction_of_the_surface():
    """many non-overlapping NPs sitting on the interface (the shell of Fig. 2): covered solid
    angle = sum of the caps"""
    rng = np.random.default_rng(5)
    pts = []
    while len(pts) < 60:
        v = rng.normal(size=3)
        v *= (R - 0.3) / np.linalg.norm(v)
        if all(np.linalg.norm(v - q) > 1.05 for q in pts):
            pts.append(v)
    m = smap(pts, [0] * 60, [0.5], W=1440, H=720) != DROP
    want = 60 * 2 * np.pi * (1 - np.cos(cap_angle(R - 0.3, 0.5)))
    assert abs(solid_angle(m) - want) < 0.05 * want
