"""Small spec builders and error norms for the tests (inputs only, no physics)."""
from __future__ import annotations

import math
import os

import numpy as np

from workloads import WorldSpec

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def quat_axis(axis: str, deg: float) -> np.ndarray:
    t = math.radians(deg) * 0.5
    c, s = math.cos(t), math.sin(t)
    return {"x": np.array([c, s, 0, 0.0]), "y": np.array([c, 0, s, 0.0]), "z": np.array([c, 0, 0, s])}[axis]


def chain_spec(n: int, total_length: float = 1.0, diameter: float = 0.05, root_quat=None,
               density: float = 800.0, E: float = 8e9, MOR: float = 60e6, apples=(),
               armature=None) -> WorldSpec:
    """n equal links in a straight line; root_quat orients the chain in the world.
    `apples` = sequence of (link, offset3, mass, k, detach)."""
    parent = np.arange(-1, n - 1, dtype=np.int32)
    length = np.full(n, total_length / n, dtype=np.float32)
    diam = np.full(n, diameter, dtype=np.float32)
    quat = np.zeros((n, 4), dtype=np.float32)
    quat[:, 0] = 1.0
    if root_quat is not None:
        q = np.asarray(root_quat, dtype=np.float64)
        quat[0] = (q / np.linalg.norm(q)).astype(np.float32)
    a = list(apples)
    return WorldSpec(
        parent=parent, length=length, diameter=diam, rest_quat=quat, density=density, E=E, MOR=MOR,
        apple_link=np.array([x[0] for x in a], dtype=np.int32),
        apple_offset=np.array([x[1] for x in a], dtype=np.float32).reshape(len(a), 3),
        apple_mass=np.array([x[2] for x in a], dtype=np.float32),
        apple_radius=np.full(len(a), 0.04, dtype=np.float32),
        apple_k=np.array([x[3] for x in a], dtype=np.float32),
        apple_detach=np.array([x[4] for x in a], dtype=np.float32),
        armature=None if armature is None else np.asarray(armature, dtype=np.float32).reshape(n, 2),
    )


def strip_apples(spec: WorldSpec) -> WorldSpec:
    import dataclasses
    z = np.zeros(0, dtype=np.float32)
    return dataclasses.replace(spec, apple_link=np.zeros(0, dtype=np.int32),
                               apple_offset=np.zeros((0, 3), dtype=np.float32), apple_mass=z, apple_radius=z,
                               apple_k=z, apple_detach=z, apple_c=None)


def rel_state_error(gpu: dict, ref: dict, x_rest: np.ndarray) -> dict:
    """Reading A27: per block B in {q, qd, x - x_rest, v}:
    |B_gpu - B_ref|_2 / max(|B_ref|_2, floor_B); floors 1e-6 sqrt(len) (q, x), 1e-4 sqrt(len) (qd, v)."""
    out = {}
    for name, floor in (("q", 1e-6), ("qd", 1e-4), ("apple_x", 1e-6), ("apple_v", 1e-4)):
        g = np.asarray(gpu[name], dtype=np.float64).ravel()
        r = np.asarray(ref[name], dtype=np.float64).ravel()
        if g.size == 0:
            out[name] = 0.0
            continue
        if name == "apple_x":
            xr = np.asarray(x_rest, dtype=np.float64).ravel()
            den = max(np.linalg.norm(r - xr), floor * math.sqrt(r.size))
        else:
            den = max(np.linalg.norm(r), floor * math.sqrt(r.size))
        out[name] = float(np.linalg.norm(g - r) / den)
    out["max"] = max(out.values())
    # Per-element view of the same comparison (not part of "max", which stays reading A27): a block 2-norm can hide one
    # badly wrong twig among 800 DoFs.  "<block>_inf" = max_j |d_j| / max(max_j |ref_j|, floor): the worst element
    # against the block's largest; "<block>_own" = max_j |d_j| / (|ref_j| + 0.01 max_j |ref_j| + floor): the worst
    # element against ITS OWN magnitude, with 1 % of the block's largest as the scale below which an element counts as
    # zero.  DESIGN.md section 5 ("Per-element bound") derives the bounds the parity tests put on them.
    for name, floor in (("q", 1e-6), ("qd", 1e-4), ("apple_x", 1e-6), ("apple_v", 1e-4)):
        g = np.asarray(gpu[name], dtype=np.float64).ravel()
        r = np.asarray(ref[name], dtype=np.float64).ravel()
        if g.size == 0:
            out[name + "_inf"] = out[name + "_own"] = 0.0
            continue
        if name == "apple_x":
            xr = np.asarray(x_rest, dtype=np.float64).ravel()
            g, r = g - xr, r - xr
        top = np.abs(r).max()
        d = np.abs(g - r)
        out[name + "_inf"] = float(d.max() / max(top, floor))
        out[name + "_own"] = float((d / (np.abs(r) + 0.01 * top + floor)).max())
    out["max_inf"] = max(out[k + "_inf"] for k in ("q", "qd", "apple_x", "apple_v"))
    out["max_own"] = max(out[k + "_own"] for k in ("q", "qd", "apple_x", "apple_v"))
    track = WORST_PER_ELEMENT.setdefault(os.environ.get("PYTEST_CURRENT_TEST", "?").split(" ")[0], {"max_inf": 0.0, "max_own": 0.0, "max": 0.0})
    for k in track:
        track[k] = max(track[k], out[k])
    return out


WORST_PER_ELEMENT: dict = {}     # test id -> worst per-element errors seen (printed by conftest at the end of the session)
