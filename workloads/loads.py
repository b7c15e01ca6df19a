"""External load schedules for BASELINE.json's configs (inputs only).

A load is a tuple (world, body, point[3], force[3]) with the semantics of
`ob_apply_wrench` (include/orchard.h): body < n_links is a link, otherwise
apple body - n_links; `point` is link-local; `force` is world-frame newtons.
"""
from __future__ import annotations

import math
from typing import List, Sequence, Tuple

import numpy as np

from .trees import MASTER_SEED, WorldSpec

Load = Tuple[int, int, Tuple[float, float, float], Tuple[float, float, float]]


def config1_loads(spec: WorldSpec, step: int, n_steps: int = 500,
                  apple_fmax: float = 30.0, branch_fmax: float = 400.0) -> List[Load]:
    """configs[0] / reading A21: at 0-based step s the ramp value is
    F_max (s+1)/n_steps; apple 0 is pulled along +x, link 4 is pulled down
    (-z) at its tip (0,0,L_4).  branch_fmax = 5000 gives config 1b (A22)."""
    f = np.float32((step + 1) / n_steps)
    fa = float(np.float32(apple_fmax) * f)
    fb = float(np.float32(branch_fmax) * f)
    n = spec.n_links
    return [
        (0, n + 0, (0.0, 0.0, 0.0), (fa, 0.0, 0.0)),
        (0, 4, (0.0, 0.0, float(spec.length[4])), (0.0, 0.0, -fb)),
    ]


def _unit_sphere(rng: np.random.Generator, size: int) -> np.ndarray:
    c = rng.uniform(-1.0, 1.0, size=size)
    psi = rng.uniform(0.0, 2.0 * math.pi, size=size)
    s = np.sqrt(np.maximum(0.0, 1.0 - c * c))
    return np.stack([s * np.cos(psi), s * np.sin(psi), c], axis=1)


def config2_pulls(specs: Sequence[WorldSpec], seed_offset: int = 2000) -> List[Load]:
    """configs[1]: from step 500 on, five random apples per world get a
    constant pull |F| ~ U(0,40) N in a uniform random direction."""
    rng = np.random.Generator(np.random.Philox(key=MASTER_SEED + seed_offset + 7))
    out: List[Load] = []
    for w, sp in enumerate(specs):
        k = min(5, sp.n_apples)
        which = np.sort(rng.choice(sp.n_apples, size=k, replace=False))
        mag = rng.uniform(0.0, 40.0, size=k)
        d = _unit_sphere(rng, k)
        for a, m, dd in zip(which, mag, d):
            f = (np.float32(m) * dd.astype(np.float32))
            out.append((w, sp.n_links + int(a), (0.0, 0.0, 0.0),
                        (float(f[0]), float(f[1]), float(f[2]))))
    return out


def wrench_process(specs: Sequence[WorldSpec], epoch: int, f_lo: float, f_hi: float,
                   seed_offset: int = 3000) -> List[Load]:
    """configs[2..4] / reading A25: one external wrench per world, resampled
    every 50 steps (epoch = step // 50): random link, random point on its
    surface, |F| ~ U(f_lo, f_hi), direction uniform on the sphere."""
    rng = np.random.Generator(np.random.Philox(key=[MASTER_SEED + seed_offset, epoch]))
    w_n = len(specs)
    u = rng.random(size=(w_n, 4))
    d = _unit_sphere(rng, w_n)
    out: List[Load] = []
    for w, sp in enumerate(specs):
        link = min(int(u[w, 0] * sp.n_links), sp.n_links - 1)
        z = float(u[w, 1]) * float(sp.length[link])
        phi = 2.0 * math.pi * float(u[w, 2])
        r = 0.5 * float(sp.diameter[link])
        mag = f_lo + float(u[w, 3]) * (f_hi - f_lo)
        f = (np.float32(mag) * d[w].astype(np.float32))
        p = np.array([r * math.cos(phi), r * math.sin(phi), z], dtype=np.float32)
        out.append((w, link, (float(p[0]), float(p[1]), float(p[2])),
                    (float(f[0]), float(f[1]), float(f[2]))))
    return out


def wrench_epoch_loads(specs: Sequence[WorldSpec], epoch: int, f_lo: float, f_hi: float,
                       seed_offset: int = 3000) -> List[Load]:
    """The A25 process as a stream of `ob_apply_wrench` calls: "resampled" means
    the wrench of epoch - 1 is withdrawn (a zero force frees its slot, reading
    A24) before the wrench of this epoch is applied, so every world carries
    exactly one external wrench at any time.  Clears come first, world by
    world, and are skipped where the new wrench lands on the same link (same
    body replaces)."""
    new = wrench_process(specs, epoch, f_lo, f_hi, seed_offset)
    if epoch == 0:
        return new
    old = wrench_process(specs, epoch - 1, f_lo, f_hi, seed_offset)
    zero = (0.0, 0.0, 0.0)
    clears = [(w, body, zero, zero) for (w, body, _p, _f), (_w, nbody, _np, _nf) in zip(old, new) if body != nbody]
    return clears + new
