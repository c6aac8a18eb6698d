"""TEST INFRASTRUCTURE -- post-processing observables of the paper, plain numpy fp64.

The paper characterises a run by statistics of the NP positions, not by trajectories
(PAPER.md:96-98): the fractal dimension (sec. 3.1, Eq. 2-4), the radial distribution
function (sec. 3.2, Eq. 6), the radial concentration profile (Eq. 8) and "aggregate
statistics" (not defined there: DESIGN.md reading R23).  Long runs of the
CUDA path and of the oracle are compared through these (tests/test_gpu_statistics.py);
nothing here is imported by the product.  Every function is the printed definition
written out -- O(N^2) where the definition is a double sum.

Pins (tests/test_oracle_observables.py): uniform points in a ball reproduce the
ball pair-distance law g(r) = 1 - 3r/(4R) + r^3/(16R^3) and C(r) = 1; a close-packed
ball of touching spheres gives D_f -> 3 with the paper's k_f = 1.593; a straight chain
has the closed-form R_g; cluster labels equal scipy's connected components.
"""
import numpy as np


def centre_of_mass(pos):
    """Eq. 4: r_0 = (1/N) sum_n r_n (identical NPs: unweighted)."""
    return np.asarray(pos, dtype=np.float64).mean(axis=0)


def radius_of_gyration(pos):
    """Eq. 3: R_g = sqrt((1/N) sum_n (r_0 - r_n)^2)."""
    x = np.asarray(pos, dtype=np.float64)
    d = x - centre_of_mass(x)
    return float(np.sqrt((d * d).sum(axis=1).mean()))


def fractal_dimension(pos, d_np, k_f=1.593):
    """Eq. 2 solved for D_f: N = k_f (2 R_g / d_NP)^D_f, with the
    paper's prefactor k_f = 1.593 (compact hexagonal structure)."""
    n = len(pos)
    return float(np.log(n / k_f) / np.log(2.0 * radius_of_gyration(pos) / d_np))


def shell_volumes(edges):
    e = np.asarray(edges, dtype=np.float64)
    return 4.0 / 3.0 * np.pi * (e[1:] ** 3 - e[:-1] ** 3)


def rdf(pos, R, dr, r_max):
    """Eq. 6: g(r) = sum_i [psi_i(r)/N] / [(N-1) dV_r / V], psi_i(r) the
    number of NPs in the shell [r, r+dr) around NP i, dV_r the shell volume and
    V = 4/3 pi R^3 the sample (droplet) volume.  As printed: no boundary correction
    (PAPER.md:139).  Returns (bin centres, g)."""
    x = np.asarray(pos, dtype=np.float64)
    n = len(x)
    nb = int(round(r_max / dr))
    edges = dr * np.arange(nb + 1)
    psi = np.zeros(nb, dtype=np.float64)          # sum over trial particles i
    for i in range(n):
        d = np.sqrt(((x - x[i]) ** 2).sum(axis=1))
        d[i] = np.inf
        psi += np.histogram(d, bins=edges)[0]
    V = 4.0 / 3.0 * np.pi * R ** 3
    g = (psi / n) / ((n - 1) * shell_volumes(edges) / V)
    return 0.5 * (edges[1:] + edges[:-1]), g


def radial_concentration(pos, R, dr):
    """Eq. 8: C(r_sun) = [psi(r_sun)/N] / [dV / V], psi the number of NPs
    in the shell [r, r+dr) around the droplet centre.  Returns (bin centres, C)."""
    x = np.asarray(pos, dtype=np.float64)
    n = len(x)
    nb = int(np.ceil(R / dr))
    edges = dr * np.arange(nb + 1)
    psi = np.histogram(np.sqrt((x * x).sum(axis=1)), bins=edges)[0].astype(np.float64)
    V = 4.0 / 3.0 * np.pi * R ** 3
    return 0.5 * (edges[1:] + edges[:-1]), (psi / n) / (shell_volumes(edges) / V)


def cluster_labels(pos, type_, sigma, bond_factor=1.5):
    """Reading R23: an aggregate is a connected component of the graph whose edges are
    the pairs with r_ij < bond_factor * sigma_ab, sigma_ab = (sigma_a + sigma_b)/2
    (1.5 sigma is the first minimum of a dense LJ g(r)).  Plain union-find over the
    O(N^2) pair list.  Returns labels in 0..n_clusters-1, numbered by first member."""
    x = np.asarray(pos, dtype=np.float64)
    t = np.asarray(type_, dtype=np.int64)
    s = np.asarray(sigma, dtype=np.float64)
    n = len(x)
    parent = np.arange(n)

    def find(a):
        while parent[a] != a:
            parent[a] = parent[parent[a]]
            a = parent[a]
        return a

    for i in range(n - 1):
        d2 = ((x[i + 1:] - x[i]) ** 2).sum(axis=1)
        lim = bond_factor * 0.5 * (s[t[i]] + s[t[i + 1:]])
        for j in np.nonzero(d2 < lim * lim)[0] + i + 1:
            a, b = find(i), find(int(j))
            if a != b:
                parent[max(a, b)] = min(a, b)
    roots = np.array([find(i) for i in range(n)])
    _, labels = np.unique(roots, return_inverse=True)
    return labels


def cluster_statistics(labels):
    """Number of aggregates, mean aggregate size (NPs per aggregate), size of the
    largest one, and the size histogram in log2 bins [1,2), [2,4), [4,8), ..."""
    sizes = np.bincount(labels)
    nb = int(np.floor(np.log2(sizes.max()))) + 1
    hist = np.bincount(np.floor(np.log2(sizes)).astype(np.int64), minlength=nb)
    return dict(n_clusters=int(len(sizes)), mean_size=float(sizes.mean()),
                largest=int(sizes.max()), log2_hist=hist)
