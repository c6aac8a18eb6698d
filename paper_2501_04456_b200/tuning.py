"""Kernel tuning choices per workload, measured on B200.  They belong
to the CUDA path, not to the inputs: `workloads.py` (the neutral module that also serves the
oracle) holds none of them."""
from __future__ import annotations

# cells per cut-off per type (lv_set_grid) measured fastest for each configuration
CELLS_PER_CUT = {
    "C1": [1], "C2": [2, 2], "C3": [1, 2, 2], "C4": [3], "C5": [1, 1],
    "T8": [1] * 8, "P1": [2], "P8": [1, 3],
}
# (skin, entries per NP) of an explicit lv_set_neighbour_list at the START of the schedule
# (the automatic setting needs neither); used by the tests that pin a fixed pool
NEIGHBOUR_LIST = {
    "C1": (0.3, 64), "C2": (0.4, 256), "C3": (0.5, 256), "C4": (0.2, 160), "C5": (0.4, 128),
    "P1": (0.3, 256), "P8": (0.4, 512),
}


def _base(w) -> str:
    return w.name.split("@")[0]


def cells_per_cut(w):
    """Tuned cells per cut-off of a workloads.Workload (scaled copies use their parent's), or None."""
    v = CELLS_PER_CUT.get(_base(w))
    return list(v) if v is not None else None


def neighbour_list(w):
    return NEIGHBOUR_LIST.get(_base(w))
