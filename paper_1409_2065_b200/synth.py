"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json `configs`).

This module holds NO arithmetic of the method (no k-NN graph, no Gaussian weights, no MM
iteration): it only draws data matrices `X`, missing-data masks and gamma grids.  It is the one
module both the oracle-side tests and the CUDA-side tests/bench may share (task rule 3).

The paper's datasets (Iris, HGDP 52 x 4,682, POPRES 370 x 10, breast cancer 84 x 9,216;
PAPER.md L148-L198) are not available; these stand in for them.  Recipes are those of
SURVEY.md 8(d) and are restated in DESIGN.md.  All arrays are drawn in fp64 from
numpy.random.default_rng(seed) and cast to fp32 ONCE, so oracle and GPU see identical values.
"""
from __future__ import annotations

import dataclasses
import numpy as np

CONFIG_NAMES = ("tiny", "expression", "genotype", "large_sparse", "dense_weight", "popres")


@dataclasses.dataclass
class Workload:
    name: str
    X: np.ndarray                # (n, p) float32, C-contiguous
    mask: np.ndarray | None      # (n, p) uint8, 1 = observed; None = all observed
    graph: str                   # "knn" or "complete"
    k: int                       # k of the k-NN graph (0 for complete graphs)
    phi_rule: str                # "fixed" or "inv_median"
    phi: float                   # value when phi_rule == "fixed"
    n_gamma: int                 # length of the gamma path
    seed: int

    @property
    def n(self) -> int:
        return int(self.X.shape[0])

    @property
    def p(self) -> int:
        return int(self.X.shape[1])


def _f32(a: np.ndarray) -> np.ndarray:
    return np.ascontiguousarray(a.astype(np.float32))


def gaussian_clusters(n, p, n_clusters, centre_sd, noise_sd, rng, outlier_frac=0.0):
    """Balanced isotropic Gaussian clusters, optional uniform outliers over the bounding box."""
    centres = rng.normal(0.0, centre_sd, size=(n_clusters, p))
    lab = np.arange(n) % n_clusters
    X = centres[lab] + rng.normal(0.0, noise_sd, size=(n, p))
    n_out = int(round(outlier_frac * n))
    if n_out:
        lo, hi = X.min(axis=0), X.max(axis=0)
        idx = rng.choice(n, size=n_out, replace=False)
        X[idx] = rng.uniform(lo, hi, size=(n_out, p))
        lab = lab.copy()
        lab[idx] = -1
    return X, lab


def make_tiny(seed=0, n=64, p=8):
    """configs[0]: 4 clusters, centres ~N(0,9I), noise sd 1; 5-NN; w=exp(-0.5 d^2); 20 gammas."""
    rng = np.random.default_rng(seed)
    X, _ = gaussian_clusters(n, p, 4, 3.0, 1.0, rng)
    return Workload("tiny", _f32(X), None, "knn", 5, "fixed", 0.5, 20, seed)


def make_expression(seed=0, n=100, p=5000, n_sub=5, block=200, shift=1.5, miss=0.10):
    """configs[1] (cf. breast cancer 84 x 9,216): N(0,1) log-expression, 5 subtypes
    each shifting the mean of its own random `block`-gene set by +-`shift`; `miss` MCAR."""
    rng = np.random.default_rng(seed)
    X = rng.normal(0.0, 1.0, size=(n, p))
    sub = np.arange(n) % n_sub
    for s in range(n_sub):
        genes = rng.choice(p, size=min(block, p), replace=False)
        sign = rng.choice([-1.0, 1.0], size=genes.size)
        X[np.ix_(sub == s, genes)] += shift * sign
    mask = (rng.random(size=(n, p)) >= miss).astype(np.uint8)
    # every column keeps at least one observed entry
    dead = np.flatnonzero(mask.sum(axis=0) == 0)
    mask[0, dead] = 1
    return Workload("expression", _f32(X), np.ascontiguousarray(mask), "knn", 10, "inv_median", 0.0, 40, seed)


def make_genotype(seed=0, n=52, p=200_000, fst=0.1, leaves=5):
    """configs[2] (cf. HGDP 52 populations): allele-frequency rows.
    Ancestral f ~ U(0.05,0.95); Balding-Nichols Beta(f(1-F)/F, (1-f)(1-F)/F) drift down a random
    `leaves`-leaf tree (root -> leaf frequencies -> population frequencies)."""
    rng = np.random.default_rng(seed)
    f0 = rng.uniform(0.05, 0.95, size=p)
    c = (1.0 - fst) / fst

    def drift(f):
        f = np.clip(f, 1e-3, 1.0 - 1e-3)
        return rng.beta(f * c, (1.0 - f) * c)

    # random tree: each leaf hangs off the root or off an earlier leaf's internal frequency
    node_f = [f0]
    leaf_f = []
    for _ in range(leaves):
        parent = node_f[int(rng.integers(0, len(node_f)))]
        child = drift(parent)
        node_f.append(child)
        leaf_f.append(child)
    pop_leaf = np.arange(n) % leaves
    X = np.empty((n, p))
    for i in range(n):
        X[i] = drift(leaf_f[pop_leaf[i]])
    return Workload("genotype", _f32(X), None, "complete", 0, "inv_median", 0.0, 50, seed)


def make_large_sparse(seed=0, n=100_000, p=64, n_clusters=50):
    """configs[3]: 50 isotropic clusters (centres ~N(0,16I), sd 1) + 2% uniform outliers; 10-NN."""
    rng = np.random.default_rng(seed)
    X, _ = gaussian_clusters(n, p, n_clusters, 4.0, 1.0, rng, outlier_frac=0.02)
    return Workload("large_sparse", _f32(X), None, "knn", 10, "inv_median", 0.0, 50, seed)


def make_dense_weight(seed=0, n=8192, p=256, n_clusters=32):
    """configs[4]: 32 Gaussian clusters, all-pairs Gaussian weights (complete graph)."""
    rng = np.random.default_rng(seed)
    X, _ = gaussian_clusters(n, p, n_clusters, 1.0, 1.0, rng)
    return Workload("dense_weight", _f32(X), None, "complete", 0, "inv_median", 0.0, 30, seed)


def make_popres(seed=0, n=3000, p=10, k=40, phi=0.0):
    """SURVEY 8(f) f3, cf. POPRES (1,896 subjects -> 370 plotted x 10 principal components,
    k = 40, phi in {0, 10}): many points, low p, large k.  A smooth cline plus weak population structure: 6 loose
    groups along a 2-D gradient embedded in p dimensions, like top principal components.  phi = 0 gives the
    uniform weights of L131."""
    rng = np.random.default_rng(seed)
    centres2 = rng.uniform(-1.0, 1.0, size=(6, 2))
    lab = np.arange(n) % 6
    xy = centres2[lab] + 0.35 * rng.normal(size=(n, 2))
    X = 0.05 * rng.normal(size=(n, p))
    X[:, :2] += xy
    X[:, 2:] *= np.linspace(1.0, 0.3, p - 2)[None, :] if p > 2 else 1.0
    return Workload("popres", _f32(X), None, "knn", k, "fixed", float(phi), 30, seed)



def side_coordinates(n: int, seed: int = 0, scale: float = 1.0):
    """Seeded GPS-like side coordinates for eq. 9: (longitude, latitude) in degrees times
    `scale`, 8 loose regional groups of which two straddle the +-180 meridian so that the modulo rule matters.
    Stand-in for the HGDP / POPRES sampling locations, which are not available.  Returns fp32 (n, 2)."""
    rng = np.random.default_rng(seed + 4242)
    lon_c = np.array([-178.0, 176.0, -120.0, -60.0, 0.0, 35.0, 90.0, 140.0])
    lat_c = rng.uniform(-50.0, 60.0, size=8)
    g = rng.integers(0, 8, size=n)
    lon = lon_c[g] + 6.0 * rng.normal(size=n)
    lon = (lon + 180.0) % 360.0 - 180.0
    lat = np.clip(lat_c[g] + 5.0 * rng.normal(size=n), -89.0, 89.0)
    return _f32(np.stack([lon, lat], axis=1) * scale)


_MAKERS = {
    "tiny": make_tiny,
    "expression": make_expression,
    "genotype": make_genotype,
    "large_sparse": make_large_sparse,
    "dense_weight": make_dense_weight,
    "popres": make_popres,
}


def make(name: str, seed: int = 0, **kw) -> Workload:
    """Build a named workload; `kw` overrides sizes (n=, p=) for reduced parity-test instances."""
    return _MAKERS[name](seed=seed, **kw)


def sample_pairs(n: int, n_pairs: int, seed: int):
    """Index pairs i<j used to estimate the median squared distance (phi rule S10): all pairs when
    there are at most `n_pairs` of them, else a seeded uniform sample.  Pure indexing, no metric."""
    total = n * (n - 1) // 2
    if total <= n_pairs:
        i, j = np.triu_indices(n, k=1)
        return i.astype(np.int64), j.astype(np.int64)
    rng = np.random.default_rng(seed + 7919)
    i = rng.integers(0, n, size=n_pairs)
    j = rng.integers(0, n - 1, size=n_pairs)
    j = j + (j >= i)
    lo, hi = np.minimum(i, j), np.maximum(i, j)
    return lo.astype(np.int64), hi.astype(np.int64)


def gamma_grid(lo: float, hi: float, n_gamma: int) -> np.ndarray:
    """Log-spaced increasing gamma path (BASELINE.json: 'log-spaced')."""
    return np.exp(np.linspace(np.log(lo), np.log(hi), n_gamma))


def tie_cases(seed: int = 0):
    """Inputs with EXACT distance ties for the k-NN tie rule (reading S9): integer lattice points (many equal
    squared distances, all exactly representable), a matrix with duplicated rows (distance 0 ties and equal
    distances to both copies), and masked lattice rows with two rows that share no observed coordinate.
    Returns a list of (name, X fp32, mask or None, k)."""
    rng = np.random.default_rng(seed + 99)
    g = np.stack(np.meshgrid(np.arange(6), np.arange(6), np.arange(3), indexing="ij"), -1).reshape(-1, 3).astype(np.float64)
    lattice = g[rng.permutation(g.shape[0])]                      # 108 points, shuffled so that index order matters
    base = rng.normal(size=(30, 5))
    dup = np.concatenate([base, base[:12], base[3:9]], axis=0)    # rows 30..41 copy 0..11, rows 42..47 copy 3..8
    dup = dup[rng.permutation(dup.shape[0])]
    lat2 = rng.integers(0, 4, size=(40, 6)).astype(np.float64)
    m2 = (rng.random(size=lat2.shape) >= 0.3).astype(np.uint8)
    m2[0, :] = [1, 1, 1, 0, 0, 0]
    m2[1, :] = [0, 0, 0, 1, 1, 1]                                 # rows 0 and 1 share no observed coordinate
    m2[2, :] = 1
    return [("lattice", _f32(lattice), None, 7), ("duplicates", _f32(dup), None, 5), ("masked_lattice", _f32(lat2), m2, 6)]


def random_graph(n: int, avg_deg: float, seed: int, connected: bool = False):
    """Seeded random undirected pair list (i<j) with uniform(0.1,1) weights, for unit tests."""
    rng = np.random.default_rng(seed)
    pairs = set()
    if connected:
        perm = rng.permutation(n)
        for a in range(1, n):
            b = int(rng.integers(0, a))
            i, j = int(perm[a]), int(perm[b])
            pairs.add((min(i, j), max(i, j)))
    target = int(avg_deg * n / 2)
    while len(pairs) < target and len(pairs) < n * (n - 1) // 2:
        i, j = int(rng.integers(0, n)), int(rng.integers(0, n))
        if i != j:
            pairs.add((min(i, j), max(i, j)))
    e = np.array(sorted(pairs), dtype=np.int32).reshape(-1, 2)
    w = rng.uniform(0.1, 1.0, size=e.shape[0])
    return e[:, 0].copy(), e[:, 1].copy(), w
