"""Thin ctypes face of liblv.so (include/lv.h): same call names, argument
marshalling only -- every step of the path runs in the library's sm_100a
kernels.  torch is used for device memory (the workspace, optional device
buffers) and for the CUDA stream; nothing else.

There is no fallback: if the library cannot be built/loaded, or there is no
CUDA device, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

from . import build as _build

MAX_TYPES = 8
SCHED_CONST, SCHED_LINEAR, SCHED_R2LAW = 0, 1, 2
WALL_ONESIDED, WALL_WINDOW = 0, 1
ST_NONFINITE, ST_OUTSIDE_GRID, ST_LIST_OVERFLOW = 1, 2, 4
DBG_KEYS, DBG_KEYS_SORTED, DBG_PERM, DBG_CELL_OFFSETS, DBG_IDS_SORTED, DBG_GRID = 1, 2, 3, 4, 5, 6
E_NONFINITE = -5
E_CAPACITY = -7
OPT_SORT, OPT_FORCE_KERNEL, OPT_TILE_SUBSTREAMS, OPT_TILE_SPAN, OPT_LIST_LANES = 1, 2, 3, 4, 5
NOALLOC_MAX_BINS = 4096          # LV_NOALLOC_MAX_BINS: bins of the static scratch of lv_observe_rdf_noalloc
E_CAPACITY = -7
SORT_COUNTING, SORT_RADIX = 0, 1
FORCE_SIMPLE, FORCE_QUEUED, FORCE_SEGMENTS, FORCE_PACKED, FORCE_TILE = 0, 1, 2, 3, 4

# every symbol include/lv.h declares (tests check the library exports them all)
SYMBOLS = ["lv_langevin_coeffs", "lv_create", "lv_set_types", "lv_set_forces",
           "lv_set_droplet_schedule", "lv_set_grid", "lv_set_option", "lv_set_neighbour_list",
           "lv_get_rebuild_count", "lv_get_list_stats", "lv_observe_rdf", "lv_observe_rdf_noalloc", "lv_observe_radial", "lv_observe_clusters", "lv_render", "lv_render_surface", "lv_workspace_bytes", "lv_bind",
           "lv_set_state", "lv_step", "lv_compute_forces", "lv_get_state", "lv_get_forces",
           "lv_get_status", "lv_get_debug", "lv_launches_per_step", "lv_step_profiled",
           "lv_stage_timing", "lv_read_stage_timing",
           "lv_measure_fp32_peak", "lv_destroy", "lv_strerror",
           "lv_last_cuda_error", "lv_version", "lv_batch_create", "lv_batch_step", "lv_batch_destroy"]


class LvView(C.Structure):
    _fields_ = [("eye_dist", C.c_double), ("focal_px", C.c_double), ("yaw", C.c_double),
                ("pitch", C.c_double), ("width", C.c_int32), ("height", C.c_int32),
                ("palette", C.c_uint32 * MAX_TYPES), ("background", C.c_uint32),
                ("droplet", C.c_uint32)]


class LvSurfaceMap(C.Structure):
    _fields_ = [("width", C.c_int32), ("height", C.c_int32),
                ("palette", C.c_uint32 * MAX_TYPES), ("droplet", C.c_uint32)]


class LvType(C.Structure):
    _fields_ = [("sigma", C.c_double), ("eps", C.c_double), ("mass", C.c_double),
                ("charge", C.c_double), ("wall_k", C.c_double), ("drag_a", C.c_double),
                ("kick_b", C.c_double)]


class GridInfo(C.Structure):
    _fields_ = [("n_types", C.c_int32), ("G", C.c_int32 * MAX_TYPES),
                ("base", C.c_uint32 * (MAX_TYPES + 1)), ("lo", C.c_float * MAX_TYPES),
                ("inv_h", C.c_float * MAX_TYPES), ("h", C.c_double * MAX_TYPES),
                ("w", C.c_int32 * (MAX_TYPES * MAX_TYPES))]


class LvError(RuntimeError):
    def __init__(self, code, what, detail=""):
        self.code = code
        super().__init__(f"{what}: {code} ({detail})")


_lib = None


def load():
    """dlopen liblv.so (building it in-tree with nvcc if it is missing or stale)."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build()
    L = C.CDLL(path)
    vp, dp, ip = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int32)
    L.lv_langevin_coeffs.argtypes = [C.c_double] * 4 + [dp, dp]
    L.lv_create.argtypes = [C.POINTER(vp), C.c_int, C.c_int, C.c_uint64, C.c_double]
    L.lv_set_types.argtypes = [vp, C.c_int, C.POINTER(LvType), dp, dp, dp, C.c_double, C.c_double]
    L.lv_set_forces.argtypes = [vp, C.c_double, dp, C.c_int]
    L.lv_set_droplet_schedule.argtypes = [vp, C.c_int, C.c_double, C.c_double, C.c_int64]
    L.lv_set_grid.argtypes = [vp, ip]
    L.lv_set_option.argtypes = [vp, C.c_int, C.c_int]
    L.lv_set_neighbour_list.argtypes = [vp, C.c_double, C.c_int]
    L.lv_get_rebuild_count.argtypes = [vp, C.POINTER(C.c_int64)]
    L.lv_get_list_stats.argtypes = [vp, C.POINTER(C.c_int64)]
    L.lv_observe_rdf.argtypes = [vp, C.c_double, C.c_int, C.POINTER(C.c_uint64), dp]
    L.lv_observe_rdf_noalloc.argtypes = [vp, C.c_double, C.c_int, C.POINTER(C.c_uint64), dp]
    L.lv_observe_clusters.argtypes = [vp, C.c_double, ip, C.POINTER(C.c_int64), dp,
                                      C.POINTER(C.c_int64), C.POINTER(C.c_uint64)]
    L.lv_render.argtypes = [vp, C.POINTER(LvView), vp, vp, C.c_int]
    L.lv_render_surface.argtypes = [vp, C.POINTER(LvSurfaceMap), vp, vp, C.c_int]
    L.lv_observe_radial.argtypes = [vp, C.c_double, C.c_int, C.POINTER(C.c_uint64), dp, dp, dp, dp,
                                    C.POINTER(C.c_int64)]
    L.lv_workspace_bytes.argtypes = [vp]
    L.lv_workspace_bytes.restype = C.c_size_t
    L.lv_bind.argtypes = [vp, vp, C.c_size_t, vp]
    L.lv_set_state.argtypes = [vp, vp, vp, vp, C.c_int64, C.c_int]
    L.lv_step.argtypes = [vp, C.c_int]
    L.lv_compute_forces.argtypes = [vp]
    L.lv_get_state.argtypes = [vp, vp, vp, vp, dp, C.POINTER(C.c_int64), C.c_int]
    L.lv_get_forces.argtypes = [vp, vp, vp, C.c_int]
    L.lv_get_status.argtypes = [vp, C.POINTER(C.c_uint32)]
    L.lv_get_debug.argtypes = [vp, C.c_int, vp, C.c_size_t, C.c_int]
    L.lv_launches_per_step.argtypes = [vp]
    L.lv_step_profiled.argtypes = [vp, C.POINTER(C.c_float)]
    L.lv_stage_timing.argtypes = [vp, C.c_int]
    L.lv_read_stage_timing.argtypes = [vp, dp, dp, C.POINTER(C.c_int64)]
    L.lv_measure_fp32_peak.argtypes = [vp, vp, dp]
    L.lv_destroy.argtypes = [vp]
    L.lv_strerror.argtypes = [C.c_int]
    L.lv_strerror.restype = C.c_char_p
    L.lv_last_cuda_error.argtypes = [vp]
    L.lv_last_cuda_error.restype = C.c_char_p
    L.lv_version.restype = C.c_char_p
    L.lv_batch_create.argtypes = [C.POINTER(vp), C.POINTER(vp), C.c_int, C.c_int]
    L.lv_batch_step.argtypes = [vp, C.c_int]
    L.lv_batch_destroy.argtypes = [vp]
    _lib = L
    return L


def langevin_coeffs(gamma, kT, mass, dt):
    a, b = C.c_double(), C.c_double()
    rc = load().lv_langevin_coeffs(gamma, kT, mass, dt, C.byref(a), C.byref(b))
    if rc != 0:
        raise LvError(rc, "lv_langevin_coeffs")
    return a.value, b.value


def _dptr(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_double))


class Batch:
    """lv_batch: bound Simulations (own streams) stepped together by one CUDA-graph launch."""

    def __init__(self, sims, steps_per_launch: int = 8):
        self.L = load()
        self.sims = list(sims)
        arr = (C.c_void_p * len(self.sims))(*[s.h for s in self.sims])
        self.h = C.c_void_p()
        rc = self.L.lv_batch_create(C.byref(self.h), arr, len(self.sims), int(steps_per_launch))
        if rc != 0:
            raise LvError(rc, "lv_batch_create", self.L.lv_strerror(rc).decode())

    def step(self, n: int = 1):
        rc = self.L.lv_batch_step(self.h, int(n))
        if rc != 0:
            raise LvError(rc, "lv_batch_step", self.L.lv_strerror(rc).decode())

    def close(self):
        if getattr(self, "h", None):
            self.L.lv_batch_destroy(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Simulation:
    """One lv_sim handle plus the torch-owned workspace and stream it uses."""

    def __init__(self, n: int, n_types: int, seed: int, dt: float, device: str = "cuda:0"):
        self.L = load()
        self.n, self.n_types = int(n), int(n_types)
        self.device = device
        self.h = C.c_void_p()
        self._check(self.L.lv_create(C.byref(self.h), self.n, self.n_types, int(seed), float(dt)),
                    "lv_create")
        self.workspace = None
        self.stream = None

    # -- errors ------------------------------------------------------------
    def _check(self, rc, what, allow=()):
        if rc != 0 and rc not in allow:
            detail = self.L.lv_strerror(rc).decode()
            if rc == -4 and self.h:
                detail += ": " + self.L.lv_last_cuda_error(self.h).decode()
            raise LvError(rc, what, detail)
        return rc

    # -- configuration (include/lv.h) ---------------------------------------
    def set_types(self, types: Sequence[dict], eps=None, sigma=None, rcut=None,
                  cut_factor: float = 2.5, coulomb_k: float = 0.0):
        arr = (LvType * self.n_types)()
        for a, t in enumerate(types):
            arr[a] = LvType(t["sigma"], t.get("eps", 1.0), t["mass"], t.get("charge", 0.0),
                            t.get("wall_k", 0.0), t.get("drag_a", 1.0), t.get("kick_b", 0.0))
        mats = [None if M is None else np.ascontiguousarray(M, dtype=np.float64).reshape(-1)
                for M in (eps, sigma, rcut)]
        self._check(self.L.lv_set_types(self.h, self.n_types, arr, _dptr(mats[0]), _dptr(mats[1]),
                                        _dptr(mats[2]), float(cut_factor), float(coulomb_k)),
                    "lv_set_types")

    def set_forces(self, g=0.0, omega2=(0.0, 0.0, 0.0), wall_mode=WALL_ONESIDED):
        o = np.asarray(omega2, dtype=np.float64)
        self._check(self.L.lv_set_forces(self.h, float(g), _dptr(o), int(wall_mode)), "lv_set_forces")

    def set_droplet_schedule(self, mode, R0, R1=None, n_steps=0):
        self._check(self.L.lv_set_droplet_schedule(self.h, int(mode), float(R0),
                                                   float(R0 if R1 is None else R1), int(n_steps)),
                    "lv_set_droplet_schedule")

    def set_grid(self, cells_per_cut):
        k = np.ascontiguousarray(cells_per_cut, dtype=np.int32)
        self._check(self.L.lv_set_grid(self.h, k.ctypes.data_as(C.POINTER(C.c_int32))), "lv_set_grid")

    def set_option(self, option: int, value: int):
        self._check(self.L.lv_set_option(self.h, int(option), int(value)), "lv_set_option")

    def set_neighbour_list(self, skin: float, capacity: int):
        self._check(self.L.lv_set_neighbour_list(self.h, float(skin), int(capacity)),
                    "lv_set_neighbour_list")

    def rebuild_count(self) -> int:
        r = C.c_int64()
        self._check(self.L.lv_get_rebuild_count(self.h, C.byref(r)), "lv_get_rebuild_count")
        return int(r.value)

    def list_stats(self) -> dict:
        o = (C.c_int64 * 6)()
        self._check(self.L.lv_get_list_stats(self.h, o), "lv_get_list_stats")
        return dict(rebuilds=int(o[0]), entries_used=int(o[1]), fallback_steps=int(o[2]), pool_entries=int(o[3]),
                    exact_rebuilds=int(o[4]), lanes_per_np=int(o[5]))

    def workspace_bytes(self) -> int:
        return int(self.L.lv_workspace_bytes(self.h))

    def bind(self, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("lv: no CUDA device -- this library has no CPU path")
        nbytes = self.workspace_bytes()
        if nbytes == 0:
            raise LvError(-2, "lv_workspace_bytes", "types/schedule not set, or CUDA unavailable")
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.Stream(device=self.device)
        ptr = (self.workspace.data_ptr() + 255) // 256 * 256
        self._check(self.L.lv_bind(self.h, ptr, nbytes, self.stream.cuda_stream), "lv_bind")

    # -- state ---------------------------------------------------------------
    @staticmethod
    def _is_torch(x):
        return hasattr(x, "data_ptr")

    def set_state(self, pos, vel, type_, step: int = 0):
        if self._is_torch(pos):
            import torch
            assert pos.is_cuda and vel.is_cuda and type_.is_cuda
            assert pos.dtype == torch.float32 and vel.dtype == torch.float32 and type_.dtype == torch.int32
            pos, vel, type_ = pos.contiguous(), vel.contiguous(), type_.contiguous()
            self.stream.wait_stream(torch.cuda.current_stream(self.device))
            rc = self.L.lv_set_state(self.h, pos.data_ptr(), vel.data_ptr(), type_.data_ptr(), int(step), 1)
            self._keep = (pos, vel, type_)
        else:
            pos = np.ascontiguousarray(pos, dtype=np.float32)
            vel = np.ascontiguousarray(vel, dtype=np.float32)
            type_ = np.ascontiguousarray(type_, dtype=np.int32)
            assert pos.shape == (self.n, 3) and vel.shape == (self.n, 3) and type_.shape == (self.n,)
            rc = self.L.lv_set_state(self.h, pos.ctypes.data, vel.ctypes.data, type_.ctypes.data, int(step), 0)
        self._check(rc, "lv_set_state")

    def set_state_ptrs(self, pos_ptr, vel_ptr, type_ptr, step, on_device):
        """Raw-pointer form (pinned host buffers in bench.py)."""
        self._check(self.L.lv_set_state(self.h, pos_ptr, vel_ptr, type_ptr, int(step), int(on_device)),
                    "lv_set_state")

    def step(self, n: int = 1):
        self._check(self.L.lv_step(self.h, int(n)), "lv_step")

    def compute_forces(self):
        self._check(self.L.lv_compute_forces(self.h), "lv_compute_forces")

    def get_state(self, on_device: bool = False, check: bool = True):
        """-> pos[n,3], vel[n,3], type[n], R, step (numpy, or torch cuda tensors)."""
        R, st = C.c_double(), C.c_int64()
        if on_device:
            import torch
            with torch.cuda.device(self.device):
                pos = torch.empty((self.n, 3), dtype=torch.float32, device=self.device)
                vel = torch.empty((self.n, 3), dtype=torch.float32, device=self.device)
                typ = torch.empty((self.n,), dtype=torch.int32, device=self.device)
            self.stream.wait_stream(torch.cuda.current_stream(self.device))
            rc = self.L.lv_get_state(self.h, pos.data_ptr(), vel.data_ptr(), typ.data_ptr(),
                                     C.byref(R), C.byref(st), 1)
        else:
            pos = np.empty((self.n, 3), dtype=np.float32)
            vel = np.empty((self.n, 3), dtype=np.float32)
            typ = np.empty((self.n,), dtype=np.int32)
            rc = self.L.lv_get_state(self.h, pos.ctypes.data, vel.ctypes.data, typ.ctypes.data,
                                     C.byref(R), C.byref(st), 0)
        self._check(rc, "lv_get_state", allow=() if check else (E_NONFINITE,))
        return pos, vel, typ, R.value, st.value

    def get_state_ptrs(self, pos_ptr, vel_ptr, type_ptr, on_device):
        R, st = C.c_double(), C.c_int64()
        self._check(self.L.lv_get_state(self.h, pos_ptr, vel_ptr, type_ptr, C.byref(R), C.byref(st),
                                        int(on_device)), "lv_get_state")
        return R.value, st.value

    def get_forces(self):
        F = np.empty((self.n, 3), dtype=np.float32)
        cnt = np.empty((self.n,), dtype=np.int32)
        self._check(self.L.lv_get_forces(self.h, F.ctypes.data, cnt.ctypes.data, 0), "lv_get_forces")
        return F, cnt

    def observe_rdf(self, dr: float, n_bins: int):
        """-> (ordered-pair counts uint64[n_bins], g[n_bins]) of Eq. 6."""
        h = np.zeros(int(n_bins), dtype=np.uint64)
        g = np.zeros(int(n_bins))
        self._check(self.L.lv_observe_rdf(self.h, float(dr), int(n_bins),
                                          h.ctypes.data_as(C.POINTER(C.c_uint64)),
                                          g.ctypes.data_as(C.POINTER(C.c_double))), "lv_observe_rdf")
        return h, g

    def observe_rdf_noalloc(self, dr: float, n_bins: int):
        """observe_rdf through the entry point whose scratch is a static device array of the
        library (no allocation, no caller scratch; n_bins <= NOALLOC_MAX_BINS)."""
        h = np.zeros(int(n_bins), dtype=np.uint64)
        g = np.zeros(int(n_bins))
        self._check(self.L.lv_observe_rdf_noalloc(self.h, float(dr), int(n_bins),
                                                  h.ctypes.data_as(C.POINTER(C.c_uint64)),
                                                  g.ctypes.data_as(C.POINTER(C.c_double))),
                    "lv_observe_rdf_noalloc")
        return h, g

    def observe_radial(self, dr: float, n_bins: int):
        """-> dict(hist, conc (Eq. 8), centre (Eq. 4), r_g (Eq. 3), d_f (Eq. 2), n_surf)."""
        h = np.zeros(int(n_bins), dtype=np.uint64)
        c = np.zeros(int(n_bins))
        ctr = np.zeros(3)
        rg, df, ns = C.c_double(), C.c_double(), C.c_int64()
        self._check(self.L.lv_observe_radial(self.h, float(dr), int(n_bins),
                                             h.ctypes.data_as(C.POINTER(C.c_uint64)),
                                             c.ctypes.data_as(C.POINTER(C.c_double)),
                                             ctr.ctypes.data_as(C.POINTER(C.c_double)),
                                             C.byref(rg), C.byref(df), C.byref(ns)),
                    "lv_observe_radial")
        return dict(hist=h, conc=c, centre=ctr, r_g=rg.value, d_f=df.value, n_surf=int(ns.value))

    def observe_clusters(self, bond_factor: float = 1.5, want_labels: bool = True):
        """-> dict(labels int32[n] by id (smallest id of the aggregate) or None, n_clusters,
        mean_size, largest, log2_hist uint64[32])."""
        lab = np.zeros(self.n, dtype=np.int32) if want_labels else None
        nc, lg, ms = C.c_int64(), C.c_int64(), C.c_double()
        hist = np.zeros(32, dtype=np.uint64)
        self._check(self.L.lv_observe_clusters(
            self.h, float(bond_factor),
            lab.ctypes.data_as(C.POINTER(C.c_int32)) if want_labels else None,
            C.byref(nc), C.byref(ms), C.byref(lg), hist.ctypes.data_as(C.POINTER(C.c_uint64))),
            "lv_observe_clusters")
        return dict(labels=lab, n_clusters=int(nc.value), mean_size=ms.value, largest=int(lg.value),
                    log2_hist=hist)

    def render(self, eye_dist, focal_px, yaw, pitch, width, height, palette,
               background=0xff000000, droplet=0xff302010, on_device=False):
        """Perspective view of the current state -> uint32[height, width] (numpy, or a torch
        tensor on the device with on_device=True)."""
        import torch
        v = LvView(float(eye_dist), float(focal_px), float(yaw), float(pitch), int(width), int(height))
        for a, c in enumerate(palette):
            v.palette[a] = int(c)
        v.background, v.droplet = int(background), int(droplet)
        with torch.cuda.device(self.device):
            n_px = int(width) * int(height)
            # depth keys (8 B per pixel) + the staged image for host output (4 B per pixel); kept
            # between calls (a fresh allocation per frame costs more than the frame)
            need = n_px + (n_px + 1) // 2
            zbuf = getattr(self, "_view_scratch", None)
            if zbuf is None or zbuf.numel() < need:
                zbuf = self._view_scratch = torch.empty(need, dtype=torch.int64, device=self.device)
            if on_device:
                img = torch.empty((int(height), int(width)), dtype=torch.int32, device=self.device)
                img.record_stream(self.stream)
                self._check(self.L.lv_render(self.h, C.byref(v), zbuf.data_ptr(), img.data_ptr(), 1),
                            "lv_render")
                return img
            img = np.zeros((int(height), int(width)), dtype=np.uint32)
            self._check(self.L.lv_render(self.h, C.byref(v), zbuf.data_ptr(), img.ctypes.data, 0),
                        "lv_render")
            self.stream.synchronize()
            return img

    def render_surface(self, width, height, palette, droplet=0xff302010, on_device=False):
        """Equirectangular map of the NP intersections with the droplet surface (Fig. 2, left
        panel) -> uint32[height, width] (numpy, or a torch tensor on the device)."""
        import torch
        m = LvSurfaceMap(int(width), int(height))
        for a, c in enumerate(palette):
            m.palette[a] = int(c)
        m.droplet = int(droplet)
        w_, h_ = max(int(width), 0), max(int(height), 0)
        with torch.cuda.device(self.device):
            need = w_ * h_ + w_ + h_ + 1 + (w_ * h_ + 1) // 2
            scratch = getattr(self, "_view_scratch", None)
            if scratch is None or scratch.numel() < need:
                scratch = self._view_scratch = torch.empty(need, dtype=torch.int64, device=self.device)
            if on_device:
                img = torch.empty((h_, w_), dtype=torch.int32, device=self.device)
                img.record_stream(self.stream)
                self._check(self.L.lv_render_surface(self.h, C.byref(m), scratch.data_ptr(),
                                                     img.data_ptr(), 1), "lv_render_surface")
                return img
            img = np.zeros((h_, w_), dtype=np.uint32)
            self._check(self.L.lv_render_surface(self.h, C.byref(m), scratch.data_ptr(),
                                                 img.ctypes.data, 0), "lv_render_surface")
            return img

    def status(self) -> int:
        s = C.c_uint32()
        self._check(self.L.lv_get_status(self.h, C.byref(s)), "lv_get_status")
        return int(s.value)

    def grid(self) -> GridInfo:
        g = GridInfo()
        self._check(self.L.lv_get_debug(self.h, DBG_GRID, C.byref(g), C.sizeof(g), 0), "lv_get_debug")
        return g

    def get_debug(self, what: int) -> np.ndarray:
        if what == DBG_CELL_OFFSETS:
            g = self.grid()
            m = int(g.base[g.n_types]) + 1
        else:
            m = self.n
        out = np.empty(m, dtype=np.uint32)
        self._check(self.L.lv_get_debug(self.h, int(what), out.ctypes.data, out.nbytes, 0), "lv_get_debug")
        return out

    def launches_per_step(self) -> int:
        return int(self.L.lv_launches_per_step(self.h))

    STAGES = ("hash", "sort", "offsets_scatter", "pair_force", "update")

    def step_profiled(self):
        """One step with per-stage CUDA-event times -> dict stage -> ms."""
        ms = (C.c_float * 5)()
        self._check(self.L.lv_step_profiled(self.h, ms), "lv_step_profiled")
        return dict(zip(self.STAGES, [float(v) for v in ms]))

    def stage_timing(self, capacity: int):
        self._check(self.L.lv_stage_timing(self.h, int(capacity)), "lv_stage_timing")

    def read_stage_timing(self):
        """-> (dict stage -> summed ms, summed step ms, steps) since the last read."""
        st = (C.c_double * 5)()
        tot, n = C.c_double(), C.c_int64()
        self._check(self.L.lv_read_stage_timing(self.h, st, C.byref(tot), C.byref(n)),
                    "lv_read_stage_timing")
        return dict(zip(self.STAGES, [float(v) for v in st])), tot.value, int(n.value)

    def measure_fp32_peak(self) -> float:
        import torch
        t = C.c_double()
        with torch.cuda.device(self.device):
            scratch = torch.empty(256, dtype=torch.uint8, device=self.device)
        self._check(self.L.lv_measure_fp32_peak(self.stream.cuda_stream, scratch.data_ptr(), C.byref(t)),
                    "lv_measure_fp32_peak")
        self.stream.synchronize()
        return t.value

    def synchronize(self):
        self.stream.synchronize()

    def close(self):
        if getattr(self, "h", None):
            self.L.lv_destroy(self.h)
            self.h = C.c_void_p()
        self.workspace = None
        self._view_scratch = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- convenience -----------------------------------------------------------
    @classmethod
    def from_workload(cls, w, cells_per_cut=None, device="cuda:0", load_state=True,
                      options=None, neighbour_list="auto") -> "Simulation":
        """Configure from a workloads.Workload: per-type (a, b) through
        lv_langevin_coeffs, Lorentz-Berthelot tables inside lv_set_types.
        neighbour_list: "auto" (default) = lv_set_neighbour_list(skin <= 0, -1), the product path
        (automatic skin and pool; the library keeps the cells below 16 384 NPs) -- unless
        `options` choose the radix sort or another force kernel than the default, which are
        cell-path choices; None = off (cells rebuilt every step); or (skin, capacity)."""
        sim = cls(w.n, w.n_types, w.seed, w.dt, device=device)
        types = []
        for a in range(w.n_types):
            da, kb = langevin_coeffs(w.gamma[a], w.kT, w.mass[a], w.dt)
            types.append(dict(sigma=w.sigma[a], eps=w.eps[a], mass=w.mass[a], charge=w.charge[a],
                              wall_k=w.wall_k[a], drag_a=da, kick_b=kb))
        sim.set_types(types, eps=w.eps_matrix, cut_factor=w.cut_factor, coulomb_k=w.coulomb_k)
        sim.set_forces(w.g, w.omega2, w.wall_mode)
        sim.set_droplet_schedule(w.sched_mode, w.R0, w.R1, w.sched_steps)
        if cells_per_cut is not None:
            sim.set_grid(cells_per_cut)
        for opt, val in (options or {}).items():
            sim.set_option(opt, val)
        if isinstance(neighbour_list, str):
            assert neighbour_list == "auto"
            o = options or {}
            cell_choice = (o.get(OPT_SORT, SORT_COUNTING) != SORT_COUNTING
                           or o.get(OPT_FORCE_KERNEL, FORCE_SEGMENTS) != FORCE_SEGMENTS)
            neighbour_list = None if cell_choice else (0.0, -1)
        if neighbour_list is not None:          # (skin, capacity)
            sim.set_neighbour_list(*neighbour_list)
        sim.bind()
        if load_state:
            sim.set_state(w.pos, w.vel, w.type, 0)
        return sim
