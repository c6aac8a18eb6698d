"""ctypes face of oracle/lv_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
`--impl reference` legs may import this package.  It imports nothing from
paper_2501_04456_b200; a workload object (from the neutral input-generator
module) is read by attribute name only.

Every function here is argument marshalling around the C functions, whose
headers cite the PAPER.md passages they follow.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

MAX_TYPES = 8

SCHED_CONST, SCHED_LINEAR, SCHED_R2LAW = 0, 1, 2
WALL_ONESIDED, WALL_WINDOW = 0, 1


class Params(C.Structure):
    _fields_ = [
        ("n_types", C.c_int32), ("wall_mode", C.c_int32), ("sched_mode", C.c_int32),
        ("pad_", C.c_int32), ("sched_steps", C.c_int64), ("seed", C.c_uint64),
        ("dt", C.c_double), ("R0", C.c_double), ("R1", C.c_double),
        ("coulomb_k", C.c_double), ("g", C.c_double), ("omega2", C.c_double * 3),
        ("sigma", C.c_double * MAX_TYPES), ("mass", C.c_double * MAX_TYPES),
        ("charge", C.c_double * MAX_TYPES), ("wall_k", C.c_double * MAX_TYPES),
        ("drag_a", C.c_double * MAX_TYPES), ("kick_b", C.c_double * MAX_TYPES),
        ("eps", C.c_double * (MAX_TYPES * MAX_TYPES)),
        ("sig", C.c_double * (MAX_TYPES * MAX_TYPES)),
        ("rcut", C.c_double * (MAX_TYPES * MAX_TYPES)),
    ]


class Grid(C.Structure):
    _fields_ = [
        ("n_types", C.c_int32), ("G", C.c_int32 * MAX_TYPES),
        ("base", C.c_uint32 * (MAX_TYPES + 1)), ("lo", C.c_float * MAX_TYPES),
        ("inv_h", C.c_float * MAX_TYPES), ("h", C.c_double * MAX_TYPES),
        ("w", C.c_int32 * (MAX_TYPES * MAX_TYPES)),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        # LV_ORACLE_LIB: another build of the same source (the sanitizer target of
        # tests/test_oracle_sanitize.py)
        path = os.environ.get("LV_ORACLE_LIB") or _build.build()
        L = C.CDLL(path)
        dp = C.POINTER(C.c_double)
        fp = C.POINTER(C.c_float)
        ip = C.POINTER(C.c_int32)
        up = C.POINTER(C.c_uint32)
        PP = C.POINTER(Params)
        GP = C.POINTER(Grid)
        L.lvo_mix_lorentz_berthelot.argtypes = [PP, dp, C.c_double]
        L.lvo_mix_lorentz_berthelot.restype = None
        L.lvo_langevin_coeffs.argtypes = [C.c_double] * 4 + [dp, dp]
        L.lvo_langevin_coeffs.restype = None
        L.lvo_radius.argtypes = [PP, C.c_int64]
        L.lvo_radius.restype = C.c_double
        for name in ("lvo_pair_forces_brute", "lvo_pair_forces_cells"):
            f = getattr(L, name)
            f.argtypes = [PP, C.c_int, dp, ip, dp, dp, ip]
            f.restype = C.c_double
        L.lvo_external_forces.argtypes = [PP, C.c_double, C.c_int, dp, ip, dp, dp]
        L.lvo_external_forces.restype = C.c_double
        L.lvo_philox4x32_10.argtypes = [up, up, up]
        L.lvo_philox4x32_10.restype = None
        L.lvo_gauss3.argtypes = [C.c_uint64, C.c_uint32, C.c_int64, dp]
        L.lvo_gauss3.restype = None
        L.lvo_gauss3_batch.argtypes = [C.c_uint64, C.c_int, up, C.c_int64, dp]
        L.lvo_gauss3_batch.restype = None
        L.lvo_step.argtypes = [PP, C.c_int, dp, dp, ip, C.c_int64, C.c_int, C.c_int, dp, dp]
        L.lvo_step.restype = C.c_int
        L.lvo_energy.argtypes = [PP, C.c_double, C.c_int, dp, dp, ip, dp]
        L.lvo_energy.restype = None
        L.lvo_grid_spec.argtypes = [PP, ip, GP]
        L.lvo_grid_spec.restype = None
        L.lvo_cell_keys.argtypes = [GP, C.c_int, fp, ip, up]
        L.lvo_cell_keys.restype = None
        L.lvo_stable_sort_perm.argtypes = [C.c_int, up, up, up]
        L.lvo_stable_sort_perm.restype = None
        L.lvo_cell_offsets.argtypes = [C.c_int, up, C.c_uint32, up]
        L.lvo_cell_offsets.restype = None
        L.lvo_rdf_hist.argtypes = [C.c_int, fp, C.c_float, C.c_int, C.POINTER(C.c_uint64)]
        L.lvo_rdf_hist.restype = None
        L.lvo_radial_hist.argtypes = [C.c_int, fp, ip, dp, C.c_double, C.c_float, C.c_int,
                                      C.POINTER(C.c_uint64), dp, C.POINTER(C.c_int64)]
        L.lvo_radial_hist.restype = None
        L.lvo_cluster_labels.argtypes = [C.c_int, fp, ip, fp, ip]
        L.lvo_cluster_labels.restype = None
        L.lvo_render.argtypes = [C.c_int, fp, ip, fp, fp, C.c_float, C.c_float, C.c_int, C.c_int, up,
                                 C.c_uint32, C.c_uint32, C.c_float, up]
        L.lvo_render.restype = None
        L.lvo_render_pixels.argtypes = L.lvo_render.argtypes
        L.lvo_render_pixels.restype = None
        L.lvo_render_surface.argtypes = [C.c_int, fp, ip, fp, C.c_float, C.c_int, C.c_int, up,
                                         C.c_uint32, up]
        L.lvo_render_surface.restype = None
        L.lvo_sizeof_params.restype = C.c_int
        L.lvo_sizeof_grid.restype = C.c_int
        L.lvo_max_threads.restype = C.c_int
        assert L.lvo_sizeof_params() == C.sizeof(Params)
        assert L.lvo_sizeof_grid() == C.sizeof(Grid)
        _lib = L
    return _lib


def _d(a):
    return a.ctypes.data_as(C.POINTER(C.c_double)) if a is not None else None


def _f(a):
    return a.ctypes.data_as(C.POINTER(C.c_float)) if a is not None else None


def _i(a):
    return a.ctypes.data_as(C.POINTER(C.c_int32)) if a is not None else None


def _u(a):
    return a.ctypes.data_as(C.POINTER(C.c_uint32)) if a is not None else None


def _c64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _ci32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def max_threads() -> int:
    return int(lib().lvo_max_threads())


def langevin_coeffs(gamma, kT, mass, dt):
    a, b = C.c_double(), C.c_double()
    lib().lvo_langevin_coeffs(gamma, kT, mass, dt, C.byref(a), C.byref(b))
    return a.value, b.value


def make_params(*, sigma, mass, charge, wall_k, drag_a, kick_b, dt, seed=0,
                eps=None, eps_matrix=None, sig_matrix=None, rcut_matrix=None,
                cut_factor=2.5, coulomb_k=0.0, g=0.0, omega2=(0.0, 0.0, 0.0),
                wall_mode=WALL_ONESIDED, sched_mode=SCHED_CONST, R0=1.0, R1=None,
                sched_steps=0) -> Params:
    """Fill a Params from physical quantities.  Pair tables: Lorentz-Berthelot
    from per-type `eps` and `cut_factor` unless explicit TxT matrices are
    given (interactions "can be freely set")."""
    T = len(sigma)
    assert 1 <= T <= MAX_TYPES
    p = Params()
    p.n_types = T
    p.wall_mode = wall_mode
    p.sched_mode = sched_mode
    p.sched_steps = int(sched_steps)
    p.seed = int(seed)
    p.dt = dt
    p.R0 = R0
    p.R1 = R0 if R1 is None else R1
    p.coulomb_k = coulomb_k
    p.g = g
    for d in range(3):
        p.omega2[d] = omega2[d]
    for a in range(T):
        p.sigma[a] = sigma[a]
        p.mass[a] = mass[a]
        p.charge[a] = charge[a]
        p.wall_k[a] = wall_k[a]
        p.drag_a[a] = drag_a[a]
        p.kick_b[a] = kick_b[a]
    e = (C.c_double * MAX_TYPES)(*([1.0] * MAX_TYPES))
    if eps is not None:
        for a in range(T):
            e[a] = eps[a]
    lib().lvo_mix_lorentz_berthelot(C.byref(p), e, cut_factor)
    for name, M in (("eps", eps_matrix), ("sig", sig_matrix), ("rcut", rcut_matrix)):
        if M is not None:
            M = np.asarray(M, dtype=np.float64).reshape(T, T)
            arr = getattr(p, name)
            for a in range(T):
                for b in range(T):
                    arr[a * MAX_TYPES + b] = M[a, b]
    return p


def params_from_workload(w) -> Params:
    """Workload (neutral input module) -> Params, using the oracle's own
    Langevin-coefficient and mixing rules."""
    ab = [langevin_coeffs(w.gamma[a], w.kT, w.mass[a], w.dt) for a in range(w.n_types)]
    return make_params(
        sigma=w.sigma, mass=w.mass, charge=w.charge, wall_k=w.wall_k,
        drag_a=[t[0] for t in ab], kick_b=[t[1] for t in ab], dt=w.dt, seed=w.seed,
        eps=w.eps, eps_matrix=w.eps_matrix, cut_factor=w.cut_factor,
        coulomb_k=w.coulomb_k, g=w.g, omega2=w.omega2, wall_mode=w.wall_mode,
        sched_mode=w.sched_mode, R0=w.R0, R1=w.R1, sched_steps=w.sched_steps)


def radius(p: Params, n: int) -> float:
    return float(lib().lvo_radius(C.byref(p), int(n)))


def pair_forces(p: Params, x, type_, method="cells"):
    """-> (F[N,3], S[N], count[N] int32, U).  method 'brute' is the definition."""
    x = _c64(x).reshape(-1, 3)
    t = _ci32(type_)
    n = x.shape[0]
    F = np.zeros((n, 3))
    S = np.zeros(n)
    cnt = np.zeros(n, dtype=np.int32)
    fn = lib().lvo_pair_forces_brute if method == "brute" else lib().lvo_pair_forces_cells
    U = fn(C.byref(p), n, _d(x), _i(t), _d(F), _d(S), _i(cnt))
    return F, S, cnt, float(U)


def external_forces(p: Params, R, x, type_):
    """-> (F[N,3], S[N], U) for wall + gravity + centrifugal at radius R."""
    x = _c64(x).reshape(-1, 3)
    t = _ci32(type_)
    n = x.shape[0]
    F = np.zeros((n, 3))
    S = np.zeros(n)
    U = lib().lvo_external_forces(C.byref(p), float(R), n, _d(x), _i(t), _d(F), _d(S))
    return F, S, float(U)


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(v) & 0xFFFFFFFF for v in ctr])
    k = (C.c_uint32 * 2)(*[int(v) & 0xFFFFFFFF for v in key])
    o = (C.c_uint32 * 4)()
    lib().lvo_philox4x32_10(c, k, o)
    return [int(v) for v in o]


def gauss3(seed, ids, step):
    ids = np.ascontiguousarray(np.asarray(ids).reshape(-1), dtype=np.uint32)
    out = np.zeros((ids.size, 3))
    lib().lvo_gauss3_batch(int(seed), ids.size, _u(ids), int(step), _d(out))
    return out


def step(p: Params, x, v, type_, step0=0, nsteps=1, method="cells", want_forces=False):
    """Advance copies of (x, v) by nsteps from step index step0.
    -> (x, v, bad) or (x, v, bad, Fpair, Fext) with the last step's forces."""
    x = _c64(x).reshape(-1, 3).copy()
    v = _c64(v).reshape(-1, 3).copy()
    t = _ci32(type_)
    n = x.shape[0]
    Fp = np.zeros((n, 3)) if want_forces else None
    Fe = np.zeros((n, 3)) if want_forces else None
    bad = lib().lvo_step(C.byref(p), n, _d(x), _d(v), _i(t), int(step0), int(nsteps),
                         0 if method == "brute" else 1, _d(Fp), _d(Fe))
    if want_forces:
        return x, v, int(bad), Fp, Fe
    return x, v, int(bad)


def energy(p: Params, R, x, v, type_):
    """-> (kinetic, pair, wall+gravity+centrifugal)."""
    x = _c64(x).reshape(-1, 3)
    v = _c64(v).reshape(-1, 3)
    t = _ci32(type_)
    out = np.zeros(3)
    lib().lvo_energy(C.byref(p), float(R), x.shape[0], _d(x), _d(v), _i(t), _d(out))
    return tuple(float(e) for e in out)


def grid_spec(p: Params, cells_per_cut=None) -> Grid:
    g = Grid()
    k = None
    if cells_per_cut is not None:
        k = (C.c_int32 * MAX_TYPES)(*([1] * MAX_TYPES))
        for a, v in enumerate(cells_per_cut):
            k[a] = int(v)
    lib().lvo_grid_spec(C.byref(p), k, C.byref(g))
    return g


def cell_structures(g: Grid, x_f32, type_):
    """fp32 positions -> (key[N], key_sorted[N], perm[N], off[n_cells+1])."""
    x = np.ascontiguousarray(x_f32, dtype=np.float32).reshape(-1, 3)
    t = _ci32(type_)
    n = x.shape[0]
    key = np.zeros(n, dtype=np.uint32)
    ks = np.zeros(n, dtype=np.uint32)
    perm = np.zeros(n, dtype=np.uint32)
    ncell = int(g.base[g.n_types])
    off = np.zeros(ncell + 1, dtype=np.uint32)
    L = lib()
    L.lvo_cell_keys(C.byref(g), n, _f(x), _i(t), _u(key))
    L.lvo_stable_sort_perm(n, _u(key), _u(ks), _u(perm))
    L.lvo_cell_offsets(n, _u(ks), ncell, _u(off))
    return key, ks, perm, off


def rdf_hist(x_f32, dr, n_bins):
    """fp32 contract #4: ordered-pair counts per shell [k dr, (k+1) dr) -> uint64[n_bins]."""
    x = np.ascontiguousarray(x_f32, dtype=np.float32).reshape(-1, 3)
    h = np.zeros(int(n_bins), dtype=np.uint64)
    inv_dr = np.float32(1.0 / float(dr))
    lib().lvo_rdf_hist(x.shape[0], _f(x), C.c_float(float(inv_dr)), int(n_bins),
                       h.ctypes.data_as(C.POINTER(C.c_uint64)))
    return h


def radial_hist(x_f32, type_, radius_a, R, dr, n_bins):
    """-> (NPs per shell around the centre uint64[n_bins], (sum x, sum y, sum z, sum |x|^2),
    N_surf)."""
    x = np.ascontiguousarray(x_f32, dtype=np.float32).reshape(-1, 3)
    t = _ci32(type_)
    ra = _c64(radius_a)
    h = np.zeros(int(n_bins), dtype=np.uint64)
    sums = np.zeros(4)
    ns = C.c_int64()
    inv_dr = np.float32(1.0 / float(dr))
    lib().lvo_radial_hist(x.shape[0], _f(x), _i(t), _d(ra), float(R), C.c_float(float(inv_dr)),
                          int(n_bins), h.ctypes.data_as(C.POINTER(C.c_uint64)), _d(sums),
                          C.byref(ns))
    return h, sums, int(ns.value)


def rdf_from_hist(hist, n, R, dr):
    """Eq. 6 from the ordered-pair counts: g_k = (psi_k / N) / ((N-1) dV_k / V)."""
    k = np.arange(len(hist), dtype=np.float64)
    dV = 4.0 / 3.0 * np.pi * (((k + 1) * dr) ** 3 - (k * dr) ** 3)
    V = 4.0 / 3.0 * np.pi * float(R) ** 3
    return (np.asarray(hist, dtype=np.float64) / n) / ((n - 1) * dV / V)


def cluster_labels(x_f32, type_, sigma_ab, bond_factor=1.5):
    """Aggregates with the bond predicate in fp32 (contract #2 with (bond_factor sigma_ab)^2):
    label[i] = smallest index of i's connected component.  sigma_ab: T x T."""
    x = np.ascontiguousarray(x_f32, dtype=np.float32).reshape(-1, 3)
    t = _ci32(type_)
    sg = np.asarray(sigma_ab, dtype=np.float64)
    rb2 = np.zeros((MAX_TYPES, MAX_TYPES), dtype=np.float32)
    T = sg.shape[0]
    rb2[:T, :T] = ((bond_factor * sg) ** 2).astype(np.float32)
    lab = np.zeros(x.shape[0], dtype=np.int32)
    lib().lvo_cluster_labels(x.shape[0], _f(x), _i(t), _f(rb2), _i(lab))
    return lab


def view_rotation(yaw, pitch):
    """Scene rotation of the headless view: pitch about x after yaw about y (fp64 -> fp32)."""
    cy, sy, cp, sp = np.cos(yaw), np.sin(yaw), np.cos(pitch), np.sin(pitch)
    return np.array([cy, 0.0, sy, sp * sy, cp, -sp * cy, -cp * sy, sp, cp * cy], dtype=np.float32)


def render(x_f32, type_, radius_a, R, eye_dist, focal_px, yaw, pitch, width, height, palette,
           background, droplet, per_pixel=False):
    """Perspective splat of Fig. 2 (right panel) -> uint32[height, width] (0xAABBGGRR).
    per_pixel: the definition written out -- every pixel against every NP (small frames)."""
    x = np.ascontiguousarray(x_f32, dtype=np.float32).reshape(-1, 3)
    t = _ci32(type_)
    ra = np.ascontiguousarray(radius_a, dtype=np.float32)
    pal = np.zeros(MAX_TYPES, dtype=np.uint32)
    pal[:len(palette)] = np.asarray(palette, dtype=np.uint32)
    rot = view_rotation(yaw, pitch)
    img = np.zeros((int(height), int(width)), dtype=np.uint32)
    fn = lib().lvo_render_pixels if per_pixel else lib().lvo_render
    fn(x.shape[0], _f(x), _i(t), _f(ra), _f(rot), C.c_float(float(np.float32(eye_dist))),
                     C.c_float(float(np.float32(focal_px))), int(width), int(height), _u(pal),
                     int(background), int(droplet), C.c_float(float(np.float32(R))), _u(img))
    return img


def render_surface(x_f32, type_, radius_a, R, width, height, palette, droplet):
    """Equirectangular map of the NP intersections with the droplet surface, Fig. 2 left panel
    (projection: this build's reading, include/lv.h) -> uint32[height, width]."""
    x = np.ascontiguousarray(x_f32, dtype=np.float32).reshape(-1, 3)
    t = _ci32(type_)
    ra = np.ascontiguousarray(radius_a, dtype=np.float32)
    pal = np.zeros(MAX_TYPES, dtype=np.uint32)
    pal[:len(palette)] = np.asarray(palette, dtype=np.uint32)
    img = np.zeros((int(height), int(width)), dtype=np.uint32)
    lib().lvo_render_surface(x.shape[0], _f(x), _i(t), _f(ra), C.c_float(float(np.float32(R))),
                             int(width), int(height), _u(pal), int(droplet), _u(img))
    return img
