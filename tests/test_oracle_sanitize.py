"""the oracle built with -fsanitize=address,undefined runs its main routes (brute
and cell pair sums, steps, cell structures, histograms, aggregates, both views) on a small mixed
system without a report.  A child process: the sanitizer runtime has to be preloaded."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

CHILD = r"""
import numpy as np
import oracle
from paper_2501_04456_b200 import workloads as W
w = W.make_workload("C3", 600)
p = oracle.params_from_workload(w)
Fb, Sb, cb, _ = oracle.pair_forces(p, w.pos, w.type, "brute")
Fc, Sc, cc, _ = oracle.pair_forces(p, w.pos, w.type, "cells")
assert np.array_equal(cb, cc)
x, v, bad = oracle.step(p, w.pos, w.vel, w.type, step0=0, nsteps=5)
assert bad == 0
g = oracle.grid_spec(p, [1, 2, 2])
oracle.cell_structures(g, w.pos, w.type)
oracle.rdf_hist(w.pos, 0.1, 40)
oracle.radial_hist(w.pos, w.type, [0.5 * s for s in w.sigma], w.R0, 0.5, 64)
sig = [[0.5 * (a + b) for b in w.sigma] for a in w.sigma]
oracle.cluster_labels(w.pos, w.type, sig, 1.5)
pal = [0x00ff8040, 0x004080ff, 0x0040ff80]
ra = [0.5 * s for s in w.sigma]
oracle.render(w.pos, w.type, ra, w.R0, 3.0 * w.R0, 60.0, 0.3, 0.2, 48, 32, pal, 0xff000000, 0xff201008)
oracle.render(w.pos, w.type, ra, w.R0, 3.0 * w.R0, 60.0, 0.3, 0.2, 24, 16, pal, 0xff000000, 0xff201008, per_pixel=True)
oracle.render_surface(w.pos, w.type, ra, w.R0, 36, 18, pal, 0xff201008)
print("sanitized oracle ok")
"""


def test_oracle_under_asan_ubsan(tmp_path):
    libasan = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    if not os.path.isabs(libasan) or not os.path.exists(libasan):
        pytest.skip("no libasan in this toolchain")
    sys.path.insert(0, ROOT)
    import oracle.build
    so = oracle.build.build_sanitized(str(tmp_path / "liblv_oracle_san.so"))
    env = dict(os.environ, LD_PRELOAD=libasan, LV_ORACLE_LIB=so, PYTHONPATH=ROOT,
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=0:exitcode=97", UBSAN_OPTIONS="halt_on_error=1:exitcode=98",
               OMP_NUM_THREADS="2")
    r = subprocess.run([sys.executable, "-c", CHILD], env=env, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, (r.stdout[-2000:], r.stderr[-4000:])
    assert "sanitized oracle ok" in r.stdout
    assert "ERROR: AddressSanitizer" not in r.stderr and "runtime error" not in r.stderr
