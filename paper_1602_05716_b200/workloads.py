"""Seeded synthetic inputs: primitive-model electrolytes in a hard-wall spherical cavity.

This module only *generates inputs* (which ions, where they start); it holds none of
the method's arithmetic, so both the CUDA path and the CPU oracle may be fed from it.
The five named workloads are the configurations of BASELINE.json; they
stand in for the paper's own runs (PAPER.md:284, 319, 351 -- primitive-model ions, N from
8192 to 1,048,576, hard-wall sphere), which used no public dataset.

Recipe: sigma = 1, l_B = 1.68 sigma, cations first then anions,
V = N sigma^3 / rho*, R = (3V / 4 pi)^(1/3); initial positions by random sequential
insertion -- each ion in array order is drawn uniformly in the ball of radius R - d/2
(uniform in the bounding cube, rejected outside the ball) and redrawn while it overlaps
an ion already placed.  Draws come from numpy's PCG64 seeded with ``seed``.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace

import numpy as np
from scipy.spatial import cKDTree


@dataclass(frozen=True)
class Species:
    count: int
    valence: float
    diameter: float


@dataclass(frozen=True)
class Workload:
    name: str
    species: tuple
    rho_star: float
    max_disp: float
    sweeps: int
    bjerrum: float = 1.68
    seed: int = 1
    hist_bin_width: float = 0.02
    hist_nbins: int = 500
    note: str = ""
    interleave: bool = False
    _cache: dict = field(default_factory=dict, compare=False, repr=False)

    @property
    def N(self) -> int:
        return sum(s.count for s in self.species)

    @property
    def cavity_R(self) -> float:
        return (3.0 * (self.N / self.rho_star) / (4.0 * math.pi)) ** (1.0 / 3.0)

    @property
    def pair_evals_per_sweep(self) -> int:
        return self.N * (self.N - 1)

    @property
    def hist_centre_rmax(self) -> float:
        """Largest centre radius such that every shell r < r_max lies inside the cavity."""
        dmax = max(s.diameter for s in self.species)
        return max(0.0, self.cavity_R - self.hist_bin_width * self.hist_nbins - 0.5 * dmax)

    def arrays(self):
        """(pos [3,N], charges [N], diameters [N]) float64; deterministic in ``seed``."""
        if "a" not in self._cache:
            q = np.concatenate([np.full(s.count, s.valence) for s in self.species]).astype(np.float64)
            d = np.concatenate([np.full(s.count, s.diameter) for s in self.species]).astype(np.float64)
            # (larger candidate batches for the million-ion system: fewer k-d tree rebuilds)
            pos = random_sequential_insertion(d, self.cavity_R, self.seed, batch=8192 if self.N <= 300000 else 131072)
            if self.interleave:
                perm = np.random.default_rng(self.seed + 7919).permutation(self.N)
                pos, q, d = pos[:, perm], q[perm], d[perm]
            self._cache["a"] = (np.ascontiguousarray(pos), q, d)
        pos, q, d = self._cache["a"]
        return pos.copy(), q.copy(), d.copy()


def random_sequential_insertion(diameters: np.ndarray, R: float, seed: int, batch: int = 8192) -> np.ndarray:
    """Place ions one after the other, uniformly in their allowed ball, no overlaps.

    Equivalent to the one-at-a-time process on the candidate stream: a candidate is kept
    iff it lies inside its ball and overlaps no earlier kept ion.  Done in batches with a
    k-d tree for speed; conflicts inside a batch are resolved in stream order.
    """
    rng = np.random.default_rng(seed)
    N = len(diameters)
    pos = np.empty((N, 3))
    placed = 0
    dmax = float(np.max(diameters))
    margin = 1.0 + 1e-12
    main_tree, main_count = None, 0
    uniform_d = bool(np.all(diameters == diameters[0]))
    guard = 0
    while placed < N:
        guard += 1
        if guard > 200000:
            raise RuntimeError("random sequential insertion did not converge (density too high)")
        d_s = float(diameters[placed])
        # run of identical diameters starting at `placed`
        run_end = placed
        while run_end < N and diameters[run_end] == d_s:
            run_end += 1
        want = run_end - placed
        a = R - 0.5 * d_s
        m = int(min(batch, max(256, 2 * want)))
        cand = (2.0 * rng.random((m, 3)) - 1.0) * a
        cand = cand[np.einsum("ij,ij->i", cand, cand) <= a * a]
        if len(cand) == 0:
            continue
        # against ions placed before this batch: a big tree rebuilt when the system has grown by
        # half, plus a small tree over the ions placed since
        if placed > 0:
            if main_tree is None or placed >= 1.5 * main_count + 64:
                main_tree, main_count = cKDTree(pos[:placed]), placed
            trees = [(main_tree, 0)]
            if placed > main_count:
                trees.append((cKDTree(pos[main_count:placed]), main_count))
            ok = np.ones(len(cand), dtype=bool)
            rmax = 0.5 * (d_s + dmax) * margin
            for tree, off in trees:
                if uniform_d:  # one diameter: the nearest neighbour decides
                    near, _ = tree.query(cand, k=1, distance_upper_bound=rmax)
                    ok &= ~np.isfinite(near)
                    continue
                kk = min(16, tree.n)  # more than can touch one sphere at these size ratios
                near, idx = tree.query(cand, k=kk, distance_upper_bound=rmax)
                near, idx = near.reshape(len(cand), kk), idx.reshape(len(cand), kk)
                found = np.isfinite(near)
                assert not found[:, -1].any() or kk == tree.n, "neighbour list truncated"
                s = 0.5 * (d_s + diameters[np.where(found, idx, 0) + off])
                ok &= ~np.any(found & (near * near < s * s * margin), axis=1)
            cand = cand[ok]
            if len(cand) == 0:
                continue
        # conflicts inside the batch, in stream order
        keep = np.ones(len(cand), dtype=bool)
        if len(cand) > 1:
            pairs = cKDTree(cand).query_pairs(r=d_s * math.sqrt(margin), output_type="ndarray")
            if len(pairs):
                pairs = pairs[np.lexsort((pairs[:, 0], pairs[:, 1]))]  # by later member, then earlier
                for a_i, b_i in pairs:  # a_i < b_i
                    if keep[a_i] and keep[b_i]:
                        keep[b_i] = False
        cand = cand[keep][:want]
        pos[placed:placed + len(cand)] = cand
        placed += len(cand)
    return np.ascontiguousarray(pos.T)


def _rpm(name, N, rho, delta, sweeps, note=""):
    return Workload(name, (Species(N // 2, +1.0, 1.0), Species(N // 2, -1.0, 1.0)), rho, delta, sweeps, note=note)


# BASELINE.json "configs", in order.  CONFIGS[3] (N = 65536) is the one the metric is quoted on.
CONFIGS = (
    _rpm("rpm_1to1_n512", 512, 0.1, 0.5, 100, "config 1: small case the oracle finishes in seconds"),
    _rpm("rpm_1to1_n4096", 4096, 0.2, 0.4, 200, "config 2"),
    Workload("asym_2to1_n16383", (Species(5461, +2.0, 1.0), Species(10922, -1.0, 0.8)), 0.25, 0.3, 100,
             note="config 3: odd N, two diameters"),
    _rpm("rpm_1to1_n65536", 65536, 0.4, 0.2, 50, "config 4: headline, g(r) 500 bins of 0.02 sigma"),
    Workload("asym_3to1_n262144", (Species(65536, +3.0, 1.2), Species(196608, -1.0, 1.0)), 0.3, 0.2, 10,
             note="config 5: oracle timed on one sweep only"),
)
HEADLINE = CONFIGS[3]


def _paper_shaped() -> Workload:
    """The paper's production system, in units of the ion diameter d = 7.5 A:
    N = 1024 x 1024 ions of a 3:-1 electrolyte, ion radius 3.75 A, Bjerrum
    length 7.117 A => l_B = 0.94893 d, bare Debye length 28.53 A = 3.804 d
    => by Eq. 5 with sum n z^2 = 3 n_total: rho* = n_total d^3 = kappa^2 / (12 pi l_B) = 1.9317e-3, R = 506.1 d;
    hard-wall sphere; trial cube of edge L/3 with L = 2R the size of the domain => max
    displacement R/3.  g(r): 500 bins of 0.1 d to 50 d = 13 Debye lengths; centres at least that far from the wall
    (the paper leaves out ions closer than 10 Debye lengths)."""
    lB = 7.117 / 7.5
    kappa = 7.5 / 28.53
    rho = kappa * kappa / (12.0 * math.pi * lB)
    N = 1024 * 1024
    R = (3.0 * (N / rho) / (4.0 * math.pi)) ** (1.0 / 3.0)
    return Workload("paper_3to1_n1048576", (Species(N // 4, +3.0, 1.0), Species(3 * N // 4, -1.0, 1.0)), rho, R / 3.0,
                    3, bjerrum=lB, hist_bin_width=0.1, hist_nbins=500,
                    note="paper-shaped production workload: N = 2^20, 3:-1, dilute, trial cube ~ L/3")


PAPER_SHAPED = _paper_shaped()
EXTRA = (PAPER_SHAPED,)


def by_name(name: str) -> Workload:
    for w in CONFIGS + EXTRA:
        if w.name == name:
            return w
    raise KeyError(name)


def scaled(base: Workload, N: int, **kw) -> Workload:
    """Same composition, density and move size as ``base`` at another N (for parity tests)."""
    tot = base.N
    counts = [max(1, round(s.count * N / tot)) for s in base.species]
    # keep charge neutrality where the base has it: fix the last species count
    zsum = sum(c * s.valence for c, s in zip(counts[:-1], base.species[:-1]))
    last = base.species[-1]
    if abs(sum(s.count * s.valence for s in base.species)) < 1e-9 and last.valence != 0:
        c_last = -zsum / last.valence
        if abs(c_last - round(c_last)) < 1e-9 and c_last > 0:
            counts[-1] = int(round(c_last))
    species = tuple(replace(s, count=c) for s, c in zip(base.species, counts))
    return replace(base, name=f"{base.name}_scaled{sum(counts)}", species=species, _cache={}, **kw)
