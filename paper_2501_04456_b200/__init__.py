"""B200-native Langevin-dynamics step for nanoparticles in an evaporating
microdroplet (arxiv 2501.04456).  The product is the C-ABI library built from
csrc/ (include/lv.h); `binding` is its thin ctypes face; `workloads` is the
neutral seeded input generator."""
__version__ = "0.1.0"
