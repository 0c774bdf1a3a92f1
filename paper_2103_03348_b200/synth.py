"""Seeded synthetic inputs for the phylogenetic-Hawkes hot path.

This module serves BOTH the CUDA path and the oracle with identical arrays and holds none of
the method's arithmetic: it only draws event locations, times and rates with the shapes of the
paper's workload (PAPER.md:194 -- 23,422 cases, 1,610 sequenced, ~700-day span, clustered
locations) following the recipe of BASELINE.json `configs` / SURVEY.md section 8(d).  The real
Ebola case files are not available; these inputs stand in for them.

Random numbers come from a self-contained counter-based generator (splitmix64 finaliser applied
to seed/stream/index), so the draws are reproducible on any machine and independent of numpy's
Generator implementation.
"""
from __future__ import annotations

import dataclasses

import numpy as np

_U64 = np.uint64
_GOLDEN = _U64(0x9E3779B97F4A7C15)


def _splitmix64(z: np.ndarray) -> np.ndarray:
    """splitmix64 output function on an array of uint64 counters (wrap-around arithmetic)."""
    with np.errstate(over="ignore"):
        z = (z + _GOLDEN).astype(_U64)
        z = ((z ^ (z >> _U64(30))) * _U64(0xBF58476D1CE4E5B9)).astype(_U64)
        z = ((z ^ (z >> _U64(27))) * _U64(0x94D049BB133111EB)).astype(_U64)
        return (z ^ (z >> _U64(31))).astype(_U64)


def uniforms(seed: int, stream: int, n: int) -> np.ndarray:
    """n uniforms in [0,1) -- (u >> 11) * 2^-53 -- from counter (seed, stream, i)."""
    with np.errstate(over="ignore"):
        base = _splitmix64(np.array([seed], dtype=_U64) * _U64(0xD1342543DE82EF95)
                           + _U64(stream) * _U64(0xA24BAED4963EE407))
        ctr = base + np.arange(n, dtype=_U64) * _GOLDEN
    u = _splitmix64(_splitmix64(ctr))
    return (u >> _U64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def normals(seed: int, stream: int, n: int) -> np.ndarray:
    """n standard normals by Box-Muller from two uniform streams."""
    u1 = uniforms(seed, 2 * stream + 1000, n)
    u2 = uniforms(seed, 2 * stream + 1001, n)
    return np.sqrt(-2.0 * np.log1p(-u1)) * np.cos(2.0 * np.pi * u2)


# Hyperparameter order everywhere: (mu0, tau_x, tau_t, xi0, h, omega)  [SURVEY.md conventions]
CONFIG_PARAMS = (0.3, 10.0, 14.0, 0.7, 1.0, 1.0 / 3.0)
# Posterior scales of PAPER.md Table 2 (tau_x=194 km, h=7.37 km, 1/omega=29.8 d); the paper has
# no tau_t (its background is space-only) so the config value is kept; weights keep
# xi0/(xi0+mu0) ~ 0.96 at the configs' overall level.
TABLE2_PARAMS = (0.04, 194.0, 14.0, 0.96, 7.37, 1.0 / 29.8)


@dataclasses.dataclass
class Events:
    """Time-sorted events.  x is SoA: x[d, i] (C-contiguous [dim, n]); theta >= 0."""
    x: np.ndarray          # [dim, n] float64
    t: np.ndarray          # [n] float64, non-decreasing
    theta: np.ndarray      # [n] float64
    free_idx: np.ndarray   # [m] int64 -- indices (in sorted order) of the events with non-unit theta
    params: tuple          # (mu0, tau_x, tau_t, xi0, h, omega)

    @property
    def n(self) -> int:
        return int(self.t.shape[0])

    @property
    def dim(self) -> int:
        return int(self.x.shape[0])


def make_events(n: int, seed: int = 0, n_centres: int | None = None, n_free: int | None = None,
                dim: int = 2, box: float = 1000.0, sigma: float = 50.0, t_max: float = 700.0,
                log_rate_sd: float = 0.5, params: tuple = CONFIG_PARAMS) -> Events:
    """BASELINE.json generator: mixture of `n_centres` isotropic Gaussian clusters (sd `sigma` km)
    with centres uniform in a `box`^dim km box; times uniform on [0, t_max] days, sorted;
    `n_free` events carry log-rate ~ N(0, log_rate_sd^2), all others theta = 1.
    Draw order (fixed): centres, assignments, offsets, times, subset, log-rates."""
    if n_centres is None:
        n_centres = max(1, int(round(60.0 * n / 23422.0)))
    if n_free is None:
        n_free = int(round(0.07 * n))
    n_free = min(n_free, n)
    centres = np.stack([uniforms(seed, 10 + d, n_centres) * box for d in range(dim)])
    assign = np.minimum((uniforms(seed, 20, n) * n_centres).astype(np.int64), n_centres - 1)
    x = np.stack([centres[d, assign] + sigma * normals(seed, 30 + d, n) for d in range(dim)])
    t = uniforms(seed, 40, n) * t_max
    order = np.argsort(t, kind="stable")
    x = np.ascontiguousarray(x[:, order])
    t = np.ascontiguousarray(t[order])
    keys = uniforms(seed, 50, n)
    free_idx = np.sort(np.argsort(keys, kind="stable")[:n_free]).astype(np.int64)
    theta = np.ones(n, dtype=np.float64)
    theta[free_idx] = np.exp(log_rate_sd * normals(seed, 60, n_free))
    return Events(x=x, t=t, theta=theta, free_idx=free_idx, params=tuple(params))


def config(idx: int, seed: int = 0, n: int | None = None) -> Events:
    """BASELINE.json `configs[idx]` inputs (idx 2/3 reuse config 1's events; idx 4 needs `n`)."""
    if idx == 0:
        return make_events(1000, seed, n_centres=20, n_free=70)
    if idx in (1, 2, 3):
        return make_events(23422, seed, n_centres=60, n_free=1610)
    if idx == 4:
        n = 50000 if n is None else n
        return make_events(n, seed)
    raise ValueError(f"no config {idx}")


def small_random(n: int, seed: int, dim: int = 2, regime: str = "mixed", ties: bool = False,
                 duplicates: bool = False) -> Events:
    """Small dense test problems whose bandwidths are comparable to the point spread, so that both
    rate components, every moment and every derivative are numerically alive (used by the finite-
    difference pins and the small parity cases)."""
    x = np.stack([uniforms(seed, 110 + d, n) * 4.0 for d in range(dim)])
    t = np.sort(uniforms(seed, 120, n) * 10.0)
    if ties and n >= 4:
        t[1] = t[2]
        t[n - 1] = t[n - 2]
        t = np.sort(t)
    if duplicates and n >= 4:
        x[:, 3] = x[:, 0]
        x[:, n - 1] = x[:, 1]
    theta = np.exp(0.5 * normals(seed, 130, n))
    if regime == "excite":
        params = (0.05, 2.0, 5.0, 0.9, 0.8, 0.7)
    elif regime == "background":
        params = (1.5, 1.5, 3.0, 0.05, 0.5, 1.2)
    else:
        params = (0.6, 1.7, 4.0, 0.5, 0.9, 0.8)
    return Events(x=np.ascontiguousarray(x), t=np.ascontiguousarray(t), theta=theta,
                  free_idx=np.arange(n, dtype=np.int64), params=params)


# ---------------------------------------------------------------------------------------------------
# Synthetic phylogeny (stands in for the 1,000 posterior trees of Dudas et al. that PAPER.md:196 uses and that
# are not in the container): a heterochronous Kingman coalescent whose tip dates are the event times of the
# sequenced subset, and a Brownian draw of the log-rates z along it.  These are INPUT draws; the density of z
# (Eq. 2) is computed by the CUDA path and, independently, by oracle/tree_ref.cpp.
@dataclasses.dataclass
class Tree:
    """2M-1 nodes; nodes 0..M-1 are the tips (tip i <-> z[i] <-> event free_idx[i]); parent[root] = -1;
    branch[v] = edge weight between v and parent[v] (branch[root] = 0)."""
    parent: np.ndarray   # [2M-1] int32
    branch: np.ndarray   # [2M-1] float64

    @property
    def n_tips(self) -> int:
        return (int(self.parent.shape[0]) + 1) // 2


def make_tree(tip_times, seed: int = 0, ne: float = 100.0, mean_root_to_tip: float = 1.0) -> Tree:
    """Coalescent backwards in time from the latest tip: with k active lineages the next merger comes after
    Exp(rate k(k-1)/(2 ne)) days; a tip joins the active set when its sampling time is passed (the waiting time is
    then redrawn).  Branch lengths (days) are finally rescaled so that the mean root-to-tip distance equals
    `mean_root_to_tip`.  Draw order: waiting times (stream 70), merging pairs (streams 71, 72)."""
    tt = np.asarray(tip_times, dtype=np.float64)
    M = int(tt.shape[0])
    if M == 1:
        return Tree(parent=np.array([-1], dtype=np.int32), branch=np.zeros(1))
    order = np.argsort(-tt, kind="stable")            # latest tip first
    u_wait = uniforms(seed, 70, 4 * M)
    u_a = uniforms(seed, 71, M)
    u_b = uniforms(seed, 72, M)
    parent = np.full(2 * M - 1, -1, dtype=np.int32)
    node_time = np.zeros(2 * M - 1)                   # backwards time (days before the latest tip)
    node_time[:M] = tt.max() - tt
    active: list[int] = []
    nxt, now, draws, merges, new_node = 0, 0.0, 0, 0, M
    while nxt < M or len(active) > 1:
        k = len(active)
        t_next_tip = node_time[order[nxt]] if nxt < M else np.inf
        if k < 2:
            now = t_next_tip
            active.append(int(order[nxt]))
            nxt += 1
            continue
        wait = -np.log1p(-u_wait[draws]) * (2.0 * ne) / (k * (k - 1.0))
        draws += 1
        if now + wait >= t_next_tip:
            now = t_next_tip
            active.append(int(order[nxt]))
            nxt += 1
            continue
        now += wait
        ia = min(int(u_a[merges] * k), k - 1)
        a = active.pop(ia)
        ib = min(int(u_b[merges] * (k - 1)), k - 2)
        b = active.pop(ib)
        merges += 1
        parent[a] = parent[b] = new_node
        node_time[new_node] = now
        active.append(new_node)
        new_node += 1
    branch = np.zeros(2 * M - 1)
    has_parent = parent >= 0
    branch[has_parent] = node_time[parent[has_parent]] - node_time[has_parent]
    # root-to-tip distances for the rescaling
    dist = np.zeros(2 * M - 1)
    for v in range(2 * M - 3, -1, -1):                # parents have larger indices than their children
        dist[v] = dist[parent[v]] + branch[v]
    branch *= mean_root_to_tip / dist[:M].mean()
    return Tree(parent=parent, branch=branch)


def draw_z(tree: Tree, sigma2: float, tau0: float, seed: int = 0) -> np.ndarray:
    """Root value ~ N(0, tau0 sigma2), each child ~ N(parent, branch sigma2); returns the tip
    values z [M].  Normal stream 80."""
    nn = int(tree.parent.shape[0])
    M = tree.n_tips
    g = normals(seed, 80, nn)
    val = np.zeros(nn)
    val[nn - 1] = np.sqrt(tau0 * sigma2) * g[nn - 1]
    for v in range(nn - 2, -1, -1):
        val[v] = val[tree.parent[v]] + np.sqrt(tree.branch[v] * sigma2) * g[v]
    return val[:M].copy()


TREE_SIGMA2, TREE_TAU0 = 0.25, 0.1


def config_tree(seed: int = 0, n: int = 23422, n_centres: int = 60, n_free: int = 1610):
    """BASELINE.json configs[2]: config 1's events, the log-rates of the `n_free` sequenced events drawn by Brownian
    diffusion (variance 0.25 per unit branch length, tau0 = 0.1) on a coalescent tree over those events' times.
    Returns (events, tree, z)."""
    ev = make_events(n, seed, n_centres=n_centres, n_free=n_free)
    tree = make_tree(ev.t[ev.free_idx], seed)
    z = draw_z(tree, TREE_SIGMA2, TREE_TAU0, seed)
    theta = np.ones(ev.n)
    theta[ev.free_idx] = np.exp(z)
    return dataclasses.replace(ev, theta=theta), tree, z
