"""Tree topologies and rest geometry for BASELINE.json's configs (inputs only).

Everything here is plain data construction: parent arrays, link lengths and
diameters, rest quaternions (child rest frame in the parent frame, Eq. 3 of the
paper), apple attachments.  No physics.

Config 1 follows SURVEY.md 8(c) readings A20-A22; the stochastic generator
follows SURVEY.md 8(d).  The paper's own generator and seed set are not
available; these stand in for them.
"""
from __future__ import annotations

import dataclasses
import math
from typing import List, Optional

import numpy as np

MASTER_SEED = 260706337


@dataclasses.dataclass
class WorldSpec:
    """One world.  All arrays are float32 / int32 so that the oracle and the
    CUDA path receive bit-identical inputs."""

    parent: np.ndarray        # [N] int32, parent[0] = -1, parent[i] < i
    length: np.ndarray        # [N] f32, m
    diameter: np.ndarray      # [N] f32, m
    rest_quat: np.ndarray     # [N,4] f32 (w,x,y,z)
    density: float
    E: float
    MOR: float
    apple_link: np.ndarray    # [A] int32
    apple_offset: np.ndarray  # [A,3] f32, link-local attach point
    apple_mass: np.ndarray    # [A] f32
    apple_radius: np.ndarray  # [A] f32
    apple_k: np.ndarray       # [A] f32
    apple_detach: np.ndarray  # [A] f32
    apple_c: Optional[np.ndarray] = None   # [A] f32 or None
    armature: Optional[np.ndarray] = None  # [N,2] f32 or None

    @property
    def n_links(self) -> int:
        return int(self.parent.shape[0])

    @property
    def n_apples(self) -> int:
        return int(self.apple_link.shape[0])


@dataclasses.dataclass
class Params:
    """Plain-data mirror of `ob_params` (include/orchard.h); defaults are the
    readings of SURVEY.md 8(c)."""

    h: float = 2e-3
    gravity: tuple = (0.0, 0.0, -9.81)
    c_d: float = 0.05
    cg_tol: float = 1e-6
    cg_max_iter: int = 200
    precond: int = 2
    cg_norm: int = 0
    rupture_frames: int = 3
    detach_frames_pull: int = 3
    detach_kappa: float = 1.1
    detach_frames_tension: int = 10
    react_max: float = 40.0
    tether_implicit: int = 1
    qd_max: float = 50.0
    zeta_s: float = 0.1
    forces_off_on_snapped: int = 1
    mass_damping: float = 0.0      # c_v = c_omega of PAPER.md:128, 1/s (reading A32); 0 = off
    fric_frac: float = 0.0         # post-rupture Coulomb friction torque as a fraction of M_max (A34); 0 = off
    fric_ramp: float = 5.0         # ... ramped up by this factor ("~5x")
    fric_time: float = 1.5         # ... over this time, s ("~1.5 s")
    fric_veps: float = 1e-2        # ... regularised below this joint speed, rad/s
    snap_drag_scale: float = 1.0   # factor on mass_damping for snapped sub-trees (A35); 1 = no reduction
    rail_speed: float = 0.0        # speed limit of the three force rails, m/s (A36); 0 = rails off
    rail_fade: float = 0.5         # power fade starts at this fraction of rail_speed
    rail_brake: float = 50.0       # speed-brake rate above rail_speed, 1/s
    range_E: tuple = (0.0, 0.0)
    range_MOR: tuple = (0.0, 0.0)
    range_density: tuple = (0.0, 0.0)
    range_detach: tuple = (0.0, 0.0)
    range_apple_mass: tuple = (0.0, 0.0)


# --------------------------------------------------------------------------
# small quaternion helpers (input construction only)
# --------------------------------------------------------------------------

def _qmul(a, b):
    aw, ax, ay, az = a
    bw, bx, by, bz = b
    return np.array([
        aw * bw - ax * bx - ay * by - az * bz,
        aw * bx + ax * bw + ay * bz - az * by,
        aw * by - ax * bz + ay * bw + az * bx,
        aw * bz + ax * by - ay * bx + az * bw,
    ], dtype=np.float64)


def _qaxis(axis: str, deg: float):
    t = math.radians(deg) * 0.5
    c, s = math.cos(t), math.sin(t)
    if axis == "x":
        return np.array([c, s, 0.0, 0.0])
    if axis == "y":
        return np.array([c, 0.0, s, 0.0])
    return np.array([c, 0.0, 0.0, s])


def _child_quat(roll_deg: float, pitch_deg: float) -> np.ndarray:
    """Rz(roll) * Rx(pitch): roll about the parent's heading, then pitch away
    from it (turtle '/' then '&')."""
    return _qmul(_qaxis("z", roll_deg), _qaxis("x", pitch_deg))


def _finish_quats(q: np.ndarray) -> np.ndarray:
    q = q / np.linalg.norm(q, axis=1, keepdims=True)
    q32 = q.astype(np.float32)
    # renormalise once in fp32 so |q|-1 is a rounding error only
    n = np.sqrt((q32.astype(np.float64) ** 2).sum(axis=1, keepdims=True))
    return (q32.astype(np.float64) / n).astype(np.float32)


# --------------------------------------------------------------------------
# config 1: deterministic binary tree of depth 4 (31 links)
# --------------------------------------------------------------------------

def binary_tree_config1() -> WorldSpec:
    """BASELINE.json configs[0]; silences filled by SURVEY.md A20/A21:
    pitch 35 deg; child c of a depth-l node has Q = Rz(137.5 l + 180 c) Rx(35);
    BFS numbering; d_c = d_p / sqrt(2); L_c = 0.8 L_p; apples on links
    15, 19, 23, 27 at the tip (0,0,L)."""
    depth = 4
    parent = [-1]
    length = [0.5]
    diam = [0.12]
    quat = [np.array([1.0, 0.0, 0.0, 0.0])]
    level_nodes = [0]
    for lvl in range(depth):
        nxt = []
        for p in level_nodes:
            for c in range(2):
                idx = len(parent)
                parent.append(p)
                length.append(0.8 * length[p])
                diam.append(diam[p] / math.sqrt(2.0))
                quat.append(_child_quat(137.5 * lvl + 180.0 * c, 35.0))
                nxt.append(idx)
        level_nodes = nxt
    n = len(parent)
    assert n == 31
    length = np.asarray(length, dtype=np.float32)
    apple_link = np.array([15, 19, 23, 27], dtype=np.int32)
    off = np.zeros((4, 3), dtype=np.float32)
    off[:, 2] = length[apple_link]
    return WorldSpec(
        parent=np.asarray(parent, dtype=np.int32),
        length=length,
        diameter=np.asarray(diam, dtype=np.float32),
        rest_quat=_finish_quats(np.asarray(quat)),
        density=800.0, E=8e9, MOR=60e6,
        apple_link=apple_link,
        apple_offset=off,
        apple_mass=np.full(4, 0.2, dtype=np.float32),
        apple_radius=np.full(4, 0.04, dtype=np.float32),
        apple_k=np.full(4, 2e3, dtype=np.float32),
        apple_detach=np.full(4, 20.0, dtype=np.float32),
    )


# --------------------------------------------------------------------------
# ternary bracketed L-system of Eq. 1: SURVEY.md 8(f) item 4
# --------------------------------------------------------------------------

def ternary_lsystem_world(n_derivations: int = 4, n_apples: int = 30,
                          rng: Optional[np.random.Generator] = None,
                          branch_angle_deg: float = 18.95, length_ratio: float = 1.109,
                          width_ratio: float = math.sqrt(3.0), f0: float = 0.22,
                          tip_diameter: float = 0.006) -> WorldSpec:
    """A -> !(v_r) F(F0) [&(a) F(F0) A] /(d1) [&(a) F(F0) A] /(d2) [&(a) F(F0) A]  from an axiom trunk,
    d1 = d2 = 137.5 deg; internodes elongate by l_r and thicken by v_r at every later derivation.
    After n derivations the body count is 1 + 2 (3^n - 1).  The paper gives no values for a, l_r, v_r, F0
    (reading A33): a = 18.95 deg and l_r = 1.109 are the classic Honda-style values of this grammar,
    v_r = sqrt(3) is the pipe rule with beta = 2 for three equal children (A20).  An internode made at
    derivation k has length F0 l_r^(n-k) and diameter tip v_r^(n-k); the axiom trunk counts as k = 0.
    Apples hang at the tips of distinct random terminal internodes."""
    n = int(n_derivations)
    rng = np.random.default_rng(0) if rng is None else rng
    parent, born, quat = [-1], [0], [np.array([1.0, 0.0, 0.0, 0.0])]
    apices = [0]                                   # internodes that carry an apex A at their tip
    for k in range(1, n + 1):
        nxt = []
        for tip in apices:
            main = len(parent)                     # F(F0): straight continuation
            parent.append(tip); born.append(k); quat.append(np.array([1.0, 0.0, 0.0, 0.0]))
            roll = 0.0
            for c in range(3):                     # [&(a) F A] /(d1) [&(a) F A] /(d2) [&(a) F A]
                parent.append(main); born.append(k); quat.append(_child_quat(roll, branch_angle_deg))
                nxt.append(len(parent) - 1)
                roll += 137.5
        apices = nxt
    N = len(parent)
    assert N == 1 + 2 * (3 ** n - 1)
    age = n - np.asarray(born)
    length = (f0 * length_ratio ** age).astype(np.float32)
    diam = (tip_diameter * width_ratio ** age).astype(np.float32)
    leaves = np.asarray(apices, dtype=np.int32)
    n_apples = min(int(n_apples), len(leaves))
    apple_link = np.sort(rng.choice(leaves, size=n_apples, replace=False)).astype(np.int32)
    off = np.zeros((n_apples, 3), dtype=np.float32)
    off[:, 2] = length[apple_link]
    return WorldSpec(
        parent=np.asarray(parent, dtype=np.int32), length=length, diameter=diam,
        rest_quat=_finish_quats(np.asarray(quat)), density=800.0, E=8e9, MOR=60e6,
        apple_link=apple_link, apple_offset=off,
        apple_mass=np.full(n_apples, 0.2, dtype=np.float32),
        apple_radius=np.full(n_apples, 0.04, dtype=np.float32),
        apple_k=np.full(n_apples, 2e3, dtype=np.float32),
        apple_detach=np.full(n_apples, 20.0, dtype=np.float32),
    )


# --------------------------------------------------------------------------
# stochastic generator (configs 2-5)
# --------------------------------------------------------------------------

def _level_widths(n_target: int, depth: int) -> List[int]:
    """W_l = round(g^l) with sum_{l<=depth} g^l = n_target; the last level
    absorbs the rounding so the widths sum to n_target."""
    lo, hi = 1.0, 8.0
    for _ in range(80):
        g = 0.5 * (lo + hi)
        s = sum(g ** l for l in range(depth + 1))
        if s < n_target:
            lo = g
        else:
            hi = g
    g = 0.5 * (lo + hi)
    w = [max(1, int(round(g ** l))) for l in range(depth + 1)]
    w[0] = 1
    w[-1] = n_target - sum(w[:-1])
    return w


def stochastic_world(rng: np.random.Generator, n_lo: int, n_hi: int, n_apples: int,
                     depth_choices=(5, 6, 7), n_target: Optional[int] = None) -> WorldSpec:
    """One stochastic bracketed-L-system-like tree.

    2-4 proposed children per node, pitch U(25,60) deg, golden-angle roll,
    length ratio U(0.7,0.9), bud abortion down to the level-width budget, pipe
    rule d_c = d_p / sqrt(#children) (beta = 2, A20).  BFS / level order,
    children of one parent contiguous.
    """
    for _attempt in range(200):
        depth = int(rng.choice(depth_choices))
        nt = int(rng.integers(n_lo, n_hi + 1)) if n_target is None else int(n_target)
        widths = _level_widths(nt, depth)
        if min(widths) < 1:
            continue
        parent = [-1]
        length = [0.5]
        diam = [float(rng.uniform(0.08, 0.15))]
        quat = [np.array([1.0, 0.0, 0.0, 0.0])]
        level_nodes = [0]
        ok = True
        for lvl in range(depth):
            budget = widths[lvl + 1]
            proposals = []  # (parent, ordinal j, pitch, ratio)
            for p in level_nodes:
                c = int(rng.integers(2, 5))
                for j in range(c):
                    proposals.append((p, j, float(rng.uniform(25.0, 60.0)),
                                      float(rng.uniform(0.7, 0.9))))
            if len(proposals) > budget:
                keep = np.sort(rng.choice(len(proposals), size=budget, replace=False))
                proposals = [proposals[k] for k in keep]
            if not proposals:
                ok = False
                break
            counts = {}
            for (p, _j, _pi, _ra) in proposals:
                counts[p] = counts.get(p, 0) + 1
            nxt = []
            for (p, j, pitch, ratio) in proposals:
                idx = len(parent)
                parent.append(p)
                length.append(length[p] * ratio)
                diam.append(diam[p] / math.sqrt(counts[p]))
                quat.append(_child_quat(137.5 * (lvl + j) + 90.0 * j, pitch))
                nxt.append(idx)
            level_nodes = nxt
        if not ok:
            continue
        n = len(parent)
        if n < n_lo or n > n_hi:
            continue
        parent_a = np.asarray(parent, dtype=np.int32)
        has_child = np.zeros(n, dtype=bool)
        has_child[parent_a[1:]] = True
        leaves = np.nonzero(~has_child)[0]
        if leaves.size < n_apples:
            continue
        apple_link = np.sort(rng.choice(leaves, size=n_apples, replace=False)).astype(np.int32)
        length_a = np.asarray(length, dtype=np.float32)
        off = np.zeros((n_apples, 3), dtype=np.float32)
        off[:, 2] = length_a[apple_link]
        return WorldSpec(
            parent=parent_a,
            length=length_a,
            diameter=np.asarray(diam, dtype=np.float32),
            rest_quat=_finish_quats(np.asarray(quat)),
            density=800.0, E=8e9, MOR=60e6,
            apple_link=apple_link,
            apple_offset=off,
            apple_mass=rng.uniform(0.15, 0.25, size=n_apples).astype(np.float32),
            apple_radius=np.full(n_apples, 0.04, dtype=np.float32),
            apple_k=np.full(n_apples, 2e3, dtype=np.float32),
            apple_detach=rng.uniform(10.0, 30.0, size=n_apples).astype(np.float32),
        )
    raise RuntimeError("stochastic_world: could not draw a tree in range")


def _rng(config: int, stream: int = 0) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=MASTER_SEED + 1000 * config + stream))


def config_params(config: int) -> Params:
    """`ob_params` for BASELINE.json configs[config-1] (1-based)."""
    dr = dict(range_E=(5e9, 11e9), range_MOR=(40e6, 80e6), range_density=(700.0, 900.0),
              range_detach=(10.0, 30.0), range_apple_mass=(0.15, 0.25))
    if config == 1:
        return Params(h=2e-3)
    if config == 2:
        return Params(h=2e-3, **dr)
    if config == 3:
        return Params(h=2e-3, **dr)
    if config == 4:
        return Params(h=1e-3, **dr)
    if config == 5:
        dr["range_MOR"] = (30e6, 60e6)
        return Params(h=1e-3, **dr)
    if config == 6:      # not a BASELINE.json config: the homogeneous ternary L-system batch of SURVEY.md 8(f) item 4
        return Params(h=1e-3, **dr)
    raise ValueError(config)


def make_config(config: int, n_worlds: Optional[int] = None) -> List[WorldSpec]:
    """World specs of BASELINE.json configs[config-1] (1-based as in SURVEY.md)."""
    if config == 1:
        return [binary_tree_config1()]
    rng = _rng(config)
    if config == 2:
        w = 64 if n_worlds is None else n_worlds
        return [stochastic_world(rng, 150, 250, 20) for _ in range(w)]
    if config in (3, 4):
        w = (1024 if config == 3 else 4096) if n_worlds is None else n_worlds
        return [stochastic_world(rng, 350, 450, 60) for _ in range(w)]
    if config == 5:
        w = 4096 if n_worlds is None else n_worlds
        out = []
        for _ in range(w):
            n = int(round(math.exp(rng.uniform(math.log(100.0), math.log(1500.0)))))
            n = min(max(n, 100), 1500)
            a = min(max(int(round(n / 10.0)), 10), 150)
            depths = (5, 6, 7, 8) if n > 600 else (5, 6, 7)
            lo, hi = max(100, n - 10), min(1500, n + 10)
            out.append(stochastic_world(rng, lo, hi, a, depth_choices=depths))
        return out
    if config == 6:      # one topology, one geometry for every world (the paper's batching model);
        w = 4096 if n_worlds is None else n_worlds   # materials and apples still differ per world (ob_randomize)
        base = ternary_lsystem_world(4, 30, rng)
        return [base for _ in range(w)]
    raise ValueError(config)
