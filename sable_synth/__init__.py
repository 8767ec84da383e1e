"""Seeded synthetic inputs for the batched AC power-flow path (SABLE, arxiv/paper_2606_07099).

This module is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA path
(`paper_2606_07099_b200/`).  It holds none of the method's arithmetic: it draws random numbers and
builds graphs.  It returns a *branch list* (from, to, r, x, b), bus types, voltage setpoints and
per-scenario net injections; admittance matrices, mismatches, Jacobians and solves are computed
separately (and independently) by the oracle and by the CUDA library.

Workloads.  The paper measures on pandapower cases 1354pegase / 3120sp / 9241pegase / ACTIVSg25k with
i.i.d. +-10 % load perturbation (eq. 20).  Those files are not available here;
BASELINE.json's five synthetic configs stand in for them.  Everything BASELINE.json states explicitly is
taken literally (bus / branch / type counts, impedance, charging and load distributions, PV share,
setpoint ranges, scaling ranges, batch sizes).  What it leaves open is read as DESIGN.md §"Input recipe"
states (reading "PA"):

* "spanning tree plus chords": preferential-attachment tree rooted at the slack (bus 0) plus
  tree-local chords (node to grandparent / sibling / uncle); no parallel branches.
* bus 0 is the slack; PV buses are a uniformly random subset of the others; setpoints are drawn once
  per network; loads sit on PQ buses only; PV generation (a fixed share of total nominal load) is split
  among PV buses with weights U(0.5, 1.5) and is not perturbed per scenario (eq. 20 perturbs
  loads only).
* `kappa` multiplies every nominal load (hence generation).  It is 1 unless the feasibility scan
  (oracle/feasibility_scan.py) found no network seed on which flat-start NR converges.

Streams: network  -> numpy Generator(PCG64(s_net)); scenarios -> PCG64(10_000 + s_net);
adjoint right-hand sides -> PCG64(20_000 + s_net).
"""
from __future__ import annotations

from dataclasses import dataclass, field
import numpy as np

PQ, PV, SLACK = 0, 1, 2


@dataclass(frozen=True)
class GridConfig:
    name: str
    n_bus: int
    n_pv: int
    n_branch: int
    r_range: tuple
    x_ratio: tuple
    b_range: tuple
    load: tuple            # ("uniform", lo, hi) or ("lognormal", mu, sigma)
    q_ratio: tuple
    gen_share: float
    vset_range: tuple
    slack_vm: float
    scale_range: tuple
    scale_per_bus: bool
    batch: int
    max_it: int
    tol: float = 1e-8
    adjoint: bool = False
    precision: int = 0     # 0 = FP64, 1 = FP64 residual + FP32 LU (Table I)
    s_net: int = 1         # accepted network seed (oracle/feasibility_scan.py)
    kappa: float = 1.0     # load scale of last resort; 1.0 = literal config


# BASELINE.json `configs`[0..4].  (config 2 lists 186 branches but "tree plus 68 chords" = 185;
# the branch count is kept, see DESIGN.md readings.)  s_net / kappa: see oracle/feasibility_scan.py.
CONFIGS = {
    1: GridConfig("cfg1_14bus", 14, 4, 20, (0.01, 0.08), (2.0, 5.0), (0.0, 0.05),
                  ("uniform", 0.05, 0.5), (0.2, 0.5), 0.60, (1.00, 1.06), 1.06,
                  (0.9, 1.1), False, 64, 20),
    2: GridConfig("cfg2_118bus", 118, 53, 186, (0.002, 0.05), (3.0, 8.0), (0.0, 0.1),
                  ("lognormal", np.log(0.3), 0.6), (0.2, 0.5), 0.70, (0.98, 1.05), 1.0,
                  (0.8, 1.2), True, 1024, 20),
    3: GridConfig("cfg3_300bus", 300, 68, 411, (0.002, 0.05), (3.0, 8.0), (0.0, 0.1),
                  ("lognormal", np.log(0.3), 0.6), (0.2, 0.5), 0.70, (0.98, 1.05), 1.0,
                  (0.85, 1.15), True, 8192, 20, adjoint=True, s_net=7, kappa=0.75),
    4: GridConfig("cfg4_2000bus", 2000, 400, 3206, (0.001, 0.03), (4.0, 10.0), (0.0, 0.08),
                  ("lognormal", np.log(0.1), 0.7), (0.2, 0.5), 0.70, (0.98, 1.05), 1.0,
                  (0.9, 1.1), True, 2048, 20, precision=1),
    5: GridConfig("cfg5_9241bus", 9241, 1444, 16049, (0.0005, 0.02), (4.0, 12.0), (0.0, 0.06),
                  ("lognormal", np.log(0.05), 0.8), (0.2, 0.5), 0.70, (0.98, 1.05), 1.0,
                  (0.95, 1.05), True, 256, 30, adjoint=True),
}


@dataclass
class Network:
    """One shared topology.  Branch k joins bus f[k] and bus t[k] (pi-model r + jx, total charging b)."""
    cfg: GridConfig
    n_bus: int
    f: np.ndarray          # int32 [n_branch]
    t: np.ndarray          # int32 [n_branch]
    r: np.ndarray          # float64 [n_branch]
    x: np.ndarray
    b: np.ndarray
    bus_type: np.ndarray   # uint8 [n_bus]: 0 = PQ, 1 = PV, 2 = slack
    slack: int
    v_set: np.ndarray      # float64 [n_bus]: |V| setpoint at PV / slack buses, 1.0 at PQ (flat start)
    p_load: np.ndarray     # nominal active load per bus (0 off PQ buses), p.u.
    q_load: np.ndarray
    p_gen: np.ndarray      # fixed active generation per bus (0 off PV buses), p.u.
    extra: dict = field(default_factory=dict)


def _pa_tree(rng: np.random.Generator, n: int) -> np.ndarray:
    """Preferential-attachment tree: node i attaches to the owner of a uniformly chosen existing
    edge end (so to node v with probability deg(v) / sum deg).  Returns parent[i], parent[0] = -1."""
    parent = np.full(n, -1, dtype=np.int64)
    ends = np.empty(2 * (n - 1), dtype=np.int64)
    m = 0
    for i in range(1, n):
        p = 0 if i == 1 else int(ends[int(rng.integers(0, m))])
        parent[i] = p
        ends[m] = p
        ends[m + 1] = i
        m += 2
    return parent


def _local_chords(rng: np.random.Generator, parent: np.ndarray, n_chords: int) -> list:
    """Tree-local chords: a random node is joined to its grandparent, a sibling, or an uncle
    (a child of its grandparent).  Duplicates, self-loops and existing tree edges are rejected."""
    n = parent.shape[0]
    children = [[] for _ in range(n)]
    for i in range(1, n):
        children[int(parent[i])].append(i)
    have = set()
    for i in range(1, n):
        a, b = i, int(parent[i])
        have.add((min(a, b), max(a, b)))
    chords = []
    tries = 0
    while len(chords) < n_chords:
        tries += 1
        if tries > 200 * (n_chords + 10):
            raise RuntimeError("chord placement failed; topology too small for the requested count")
        v = int(rng.integers(1, n))
        kind = int(rng.integers(0, 3))
        p = int(parent[v])
        gp = int(parent[p]) if p >= 0 else -1
        if kind == 0:
            w = gp
        elif kind == 1:
            sib = children[p]
            w = sib[int(rng.integers(0, len(sib)))] if len(sib) > 1 else -1
        else:
            unc = children[gp] if gp >= 0 else []
            w = unc[int(rng.integers(0, len(unc)))] if len(unc) > 1 else -1
        if w < 0 or w == v:
            continue
        key = (min(v, w), max(v, w))
        if key in have:
            continue
        have.add(key)
        chords.append(key)
    return chords


def make_network(cfg_id: int | GridConfig, s_net: int | None = None, kappa: float | None = None) -> Network:
    cfg = CONFIGS[cfg_id] if not isinstance(cfg_id, GridConfig) else cfg_id
    s_net = cfg.s_net if s_net is None else s_net
    kappa = cfg.kappa if kappa is None else kappa
    rng = np.random.Generator(np.random.PCG64(s_net))
    n = cfg.n_bus
    parent = _pa_tree(rng, n)
    chords = _local_chords(rng, parent, cfg.n_branch - (n - 1))
    f = np.concatenate([np.arange(1, n, dtype=np.int64), np.array([c[0] for c in chords], dtype=np.int64)])
    t = np.concatenate([parent[1:], np.array([c[1] for c in chords], dtype=np.int64)])
    nb = f.shape[0]
    assert nb == cfg.n_branch
    r = rng.uniform(cfg.r_range[0], cfg.r_range[1], nb)
    x = r * rng.uniform(cfg.x_ratio[0], cfg.x_ratio[1], nb)
    b = rng.uniform(cfg.b_range[0], cfg.b_range[1], nb)

    bus_type = np.zeros(n, dtype=np.uint8)
    bus_type[0] = SLACK
    pv = rng.choice(np.arange(1, n), size=cfg.n_pv, replace=False)
    bus_type[pv] = PV
    v_set = np.ones(n)
    v_set[0] = cfg.slack_vm
    v_set[np.sort(pv)] = rng.uniform(cfg.vset_range[0], cfg.vset_range[1], cfg.n_pv)

    pq = np.flatnonzero(bus_type == PQ)
    if cfg.load[0] == "uniform":
        pl = rng.uniform(cfg.load[1], cfg.load[2], pq.shape[0])
    else:
        pl = rng.lognormal(cfg.load[1], cfg.load[2], pq.shape[0])
    ql = pl * rng.uniform(cfg.q_ratio[0], cfg.q_ratio[1], pq.shape[0])
    p_load = np.zeros(n)
    q_load = np.zeros(n)
    p_load[pq] = kappa * pl
    q_load[pq] = kappa * ql
    w = rng.uniform(0.5, 1.5, cfg.n_pv)
    p_gen = np.zeros(n)
    if cfg.n_pv:
        p_gen[np.sort(pv)] = cfg.gen_share * p_load.sum() * w / w.sum()
    return Network(cfg, n, f.astype(np.int32), t.astype(np.int32), r, x, b, bus_type, 0, v_set,
                   p_load, q_load, p_gen, {"s_net": s_net, "kappa": kappa, "parent": parent})


def make_scenarios(net: Network, batch: int | None = None, seed: int | None = None):
    """Per-scenario net injections (P_spec = p_g - p_d) and setpoints.

    Returns p_spec, q_spec, v_set, each float64 [batch][n_bus], C-contiguous.  Loads are scaled by one
    factor per scenario (config 1) or per (scenario, bus) (configs 2-5), applied to P and Q alike."""
    cfg = net.cfg
    batch = cfg.batch if batch is None else batch
    seed = 10_000 + net.extra["s_net"] if seed is None else seed
    rng = np.random.Generator(np.random.PCG64(seed))
    lo, hi = cfg.scale_range
    if cfg.scale_per_bus:
        s = rng.uniform(lo, hi, (batch, net.n_bus))
    else:
        s = np.repeat(rng.uniform(lo, hi, (batch, 1)), net.n_bus, axis=1)
    p_spec = net.p_gen[None, :] - s * net.p_load[None, :]
    q_spec = -s * net.q_load[None, :]
    v_set = np.repeat(net.v_set[None, :], batch, axis=0)
    return (np.ascontiguousarray(p_spec), np.ascontiguousarray(q_spec), np.ascontiguousarray(v_set))


def make_adjoint_rhs(net: Network, batch: int | None = None, seed: int | None = None):
    """g ~ N(0, 1) on every theta / V_m unknown (BASELINE.json config 3), zero elsewhere.

    Returns g_va, g_vm float64 [batch][n_bus]: g_va is zero at the slack, g_vm is zero off PQ buses."""
    batch = net.cfg.batch if batch is None else batch
    seed = 20_000 + net.extra["s_net"] if seed is None else seed
    rng = np.random.Generator(np.random.PCG64(seed))
    g_va = rng.standard_normal((batch, net.n_bus))
    g_vm = rng.standard_normal((batch, net.n_bus))
    g_va[:, net.bus_type == SLACK] = 0.0
    g_vm[:, net.bus_type != PQ] = 0.0
    return np.ascontiguousarray(g_va), np.ascontiguousarray(g_vm)


def tiny_network(n_bus: int, n_extra: int, n_pv: int, seed: int, load=(0.05, 0.3)) -> Network:
    """Small random networks for property tests (any size >= 2); same recipe as config 1."""
    cfg = GridConfig(f"tiny{n_bus}_{seed}", n_bus, n_pv, n_bus - 1 + n_extra, (0.01, 0.08), (2.0, 5.0),
                     (0.0, 0.05), ("uniform", load[0], load[1]), (0.2, 0.5), 0.6 if n_pv else 0.0,
                     (1.00, 1.06), 1.04, (0.9, 1.1), True, 8, 20)
    return make_network(cfg, s_net=seed, kappa=1.0)


def standin_config(n_bus: int, batch: int = 256) -> GridConfig:
    """Paper-shaped stand-ins: synthetic grids of the sizes of the paper's cases
    (1 354 / 3 120 / 9 241 / 25 000 buses) drawn by the recipe above with +-10 % i.i.d. load
    perturbation per scenario and load (eq. 20).  Nothing of the pandapower case files is reproduced."""
    big = n_bus > 5000
    return GridConfig(name=f"standin{n_bus}", n_bus=n_bus, n_pv=int(round(0.18 * n_bus)), n_branch=int(round(1.6 * n_bus)),
                      r_range=(0.0005, 0.02) if big else (0.001, 0.03), x_ratio=(4.0, 12.0) if big else (4.0, 10.0),
                      b_range=(0.0, 0.06), load=("lognormal", float(np.log(0.05 if big else 0.1)), 0.8 if big else 0.7),
                      q_ratio=(0.2, 0.5), gen_share=0.7, vset_range=(0.98, 1.05), slack_vm=1.0, scale_range=(0.9, 1.1),
                      scale_per_bus=True, batch=batch, max_it=30)


def mesh_network(nx: int, ny: int, seed: int = 1, kappa: float = 0.3, n_pv_frac: float = 0.15, batch: int = 512) -> Network:
    """Higher-fill stand-in: an nx x ny lattice (every bus joined to its right and lower neighbour) with a fraction of
    the lattice edges removed at random while keeping the graph connected, plus a few diagonal ties.  Minimum-degree
    fill on such meshes is 2-4x nnz(J1) (transmission grids sit between this and the tree-like configs 1-5), so the
    launch policy is exercised away from its low-fill tuning points.  Same impedance / load recipe as config 4;
    `kappa` scales the loads so that the flat start converges (meshes of long lines are weak)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    n = nx * ny
    idx = lambda i, j: i * ny + j
    edges = []
    for i in range(nx):
        for j in range(ny):
            if j + 1 < ny:
                edges.append((idx(i, j), idx(i, j + 1)))
            if i + 1 < nx:
                edges.append((idx(i, j), idx(i + 1, j)))
    edges = [edges[k] for k in rng.permutation(len(edges))]
    # spanning tree first (union-find), then 70 % of the remaining lattice edges, then n/20 diagonal ties
    root = list(range(n))

    def find(a):
        while root[a] != a:
            root[a] = root[root[a]]
            a = root[a]
        return a
    tree, rest = [], []
    for a, b in edges:
        ra, rb = find(a), find(b)
        if ra != rb:
            root[ra] = rb
            tree.append((a, b))
        else:
            rest.append((a, b))
    keep = tree + rest[: int(0.7 * len(rest))]
    have = set((min(a, b), max(a, b)) for a, b in keep)
    for _ in range(n // 20):
        i, j = int(rng.integers(0, nx - 1)), int(rng.integers(0, ny - 1))
        e = (idx(i, j), idx(i + 1, j + 1))
        if e not in have:
            have.add(e)
            keep.append(e)
    n_pv = int(round(n_pv_frac * n))
    cfg = GridConfig(name=f"mesh{nx}x{ny}", n_bus=n, n_pv=n_pv, n_branch=len(keep), r_range=(0.001, 0.03), x_ratio=(4.0, 10.0),
                     b_range=(0.0, 0.08), load=("lognormal", float(np.log(0.1)), 0.7), q_ratio=(0.2, 0.5), gen_share=0.7,
                     vset_range=(0.98, 1.05), slack_vm=1.0, scale_range=(0.9, 1.1), scale_per_bus=True, batch=batch, max_it=20,
                     s_net=seed, kappa=kappa)
    f = np.array([e[0] for e in keep], dtype=np.int64)
    t = np.array([e[1] for e in keep], dtype=np.int64)
    nb = f.shape[0]
    r = rng.uniform(cfg.r_range[0], cfg.r_range[1], nb)
    x = r * rng.uniform(cfg.x_ratio[0], cfg.x_ratio[1], nb)
    b = rng.uniform(cfg.b_range[0], cfg.b_range[1], nb)
    bus_type = np.zeros(n, dtype=np.uint8)
    slack = idx(nx // 2, ny // 2)
    bus_type[slack] = SLACK
    others = np.array([i for i in range(n) if i != slack])
    pv = rng.choice(others, size=n_pv, replace=False)
    bus_type[pv] = PV
    v_set = np.ones(n)
    v_set[np.sort(pv)] = rng.uniform(cfg.vset_range[0], cfg.vset_range[1], n_pv)
    pq = np.flatnonzero(bus_type == PQ)
    pl = rng.lognormal(cfg.load[1], cfg.load[2], pq.shape[0])
    ql = pl * rng.uniform(cfg.q_ratio[0], cfg.q_ratio[1], pq.shape[0])
    p_load = np.zeros(n); q_load = np.zeros(n)
    p_load[pq] = kappa * pl; q_load[pq] = kappa * ql
    w = rng.uniform(0.5, 1.5, n_pv)
    p_gen = np.zeros(n)
    p_gen[np.sort(pv)] = cfg.gen_share * p_load.sum() * w / w.sum()
    return Network(cfg, n, f.astype(np.int32), t.astype(np.int32), r, x, b, bus_type, int(slack), v_set, p_load, q_load, p_gen,
                   {"s_net": seed, "kappa": kappa})


def ybus_triplets(n_bus, f, t, r, x, b):
    """Harness-side input preparation for the CUDA library only (the oracle assembles its own Y_bus in C and never calls
    this): the pi-model branch list as Y_bus CSR triplets -- unsorted, with duplicates, which sable_create canonicalises.
    The paper takes Y_bus as given.  Returns (row_ptr, col, G, B)."""
    f = np.asarray(f, np.int64); t = np.asarray(t, np.int64)
    y = 1.0 / (np.asarray(r, float) + 1j * np.asarray(x, float))
    sh = 0.5j * np.asarray(b, float)
    rows = np.concatenate([f, t, f, t]); cols = np.concatenate([f, t, t, f])
    vals = np.concatenate([y + sh, y + sh, -y, -y])
    order = np.argsort(rows, kind="stable")
    rows, cols, vals = rows[order], cols[order], vals[order]
    row_ptr = np.zeros(n_bus + 1, np.int64)
    np.add.at(row_ptr, rows + 1, 1)
    row_ptr = np.cumsum(row_ptr).astype(np.int32)
    return row_ptr, cols.astype(np.int32), np.ascontiguousarray(vals.real), np.ascontiguousarray(vals.imag)
