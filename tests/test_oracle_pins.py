"""Pins for the fp64 oracle: closed forms, invariants,
hand-derived Lagrangian dynamics and brute force, none of which call back into
the oracle's own formulas.  CPU only."""
from __future__ import annotations

import dataclasses
import math
import os

import numpy as np
import pytest
import scipy.linalg
from scipy.spatial.transform import Rotation

from helpers import GOLDEN, chain_spec, quat_axis, strip_apples
from oracle import OracleWorld, philox4x32_10
from workloads import Params, binary_tree_config1, config1_loads, config_params, stochastic_world

G = float(np.float32(9.81))      # the fp32 value both implementations receive


def _level_of(parent):
    lv = np.zeros(len(parent), dtype=int)
    for i in range(1, len(parent)):
        lv[i] = lv[parent[i]] + 1
    return lv


# ---------------------------------------------------------------- P12 Philox
def test_philox_known_answers():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "philox4x32_10_kat.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        out = philox4x32_10(v[0:4], v[4:6])
        assert [int(x) for x in out] == v[6:10]


def test_philox_bijection_and_uniformity():
    # a counter-based generator is a bijection of the counter for a fixed key
    key = [0x1234, 0x5678]
    outs = {tuple(int(x) for x in philox4x32_10([i, 0, 0, 0], key)) for i in range(2000)}
    assert len(outs) == 2000
    u = np.array([philox4x32_10([i, 3, 1, 0], key)[0] >> 8 for i in range(4000)], dtype=np.float64) / 2 ** 24
    assert abs(u.mean() - 0.5) < 0.02 and abs(u.var() - 1 / 12) < 0.01


def test_randomize_draws_follow_reading_A23():
    spec = binary_tree_config1()
    P = config_params(2)
    w = OracleWorld(spec, P, world_index=7)
    seed = 0x0123456789ABCDEF
    w.randomize(seed)
    key = [seed & 0xFFFFFFFF, seed >> 32]
    o = philox4x32_10([7, 0, 0, 0], key)

    def uni(x, lo, hi):
        u = np.float32(int(x) >> 8) * np.float32(2.0 ** -24)
        # fmaf in fp32: a double product/sum of fp32 operands is exact before the single rounding
        return np.float32(np.float64(u) * np.float64(np.float32(hi) - np.float32(lo)) + np.float64(np.float32(lo)))
    mat = w.material()
    assert mat["E"] == uni(o[0], *P.range_E)
    assert mat["MOR"] == uni(o[1], *P.range_MOR)
    assert mat["density"] == uni(o[2], *P.range_density)
    for a in range(spec.n_apples):
        oa = philox4x32_10([7, a, 1, 0], key)
        assert np.float32(mat["detach"][a]) == uni(oa[0], *P.range_detach)
        assert np.float32(mat["mass"][a]) == uni(oa[1], *P.range_apple_mass)
    assert P.range_E[0] <= mat["E"] <= P.range_E[1]
    # degenerate ranges keep the spec
    w2 = OracleWorld(spec, config_params(1), world_index=7)
    w2.randomize(seed)
    m2 = w2.material()
    assert m2["E"] == np.float32(8e9) and m2["MOR"] == np.float32(60e6) and m2["density"] == np.float32(800.0)
    assert np.allclose(m2["detach"], 20.0) and np.allclose(m2["mass"], 0.2)


# ---------------------------------------------------------------- P1 constants
def test_config1_closed_form_constants():
    spec = binary_tree_config1()
    w = OracleWorld(spec, config_params(1))
    d = w.derived()
    lv = _level_of(spec.parent)
    rows = [l.split() for l in open(os.path.join(GOLDEN, "config1_closed_forms.txt")) if l.strip() and l[0] != "#"]
    for r in rows:
        level, K, Mmax, m = int(r[0]), float(r[1]), float(r[2]), float(r[3])
        idx = np.nonzero(lv == level)[0]
        assert idx.size == 2 ** level
        # fp32 inputs (d, L) carry ~1e-7 relative error; the printed values carry 4-6 digits
        assert np.all(np.abs(d["K"][idx] - K) <= 0.5 + 1e-5 * K)
        assert np.all(np.abs(d["Mmax"][idx] - Mmax) <= 0.5)
        assert np.all(np.abs(d["m"][idx] - m) <= 0.0005)
    # r-form of Eq. 4 / Eq. 5 (the oracle uses the d-form, reading A31)
    r = spec.diameter.astype(np.float64) / 2
    L = spec.length.astype(np.float64)
    assert np.allclose(d["K"], math.pi / 4 * 8e9 * r ** 4 / L, rtol=1e-12)
    assert np.allclose(d["Mmax"], 60e6 * math.pi * r ** 3 / 4, rtol=1e-12)
    # cylinder inertia about its centre (textbook)
    assert np.allclose(d["Ixx"], d["m"] * (3 * r * r + L * L) / 12, rtol=1e-12)
    assert np.allclose(d["Izz"], d["m"] * r * r / 2, rtol=1e-12)


# ---------------------------------------------------------------- FK vs scipy
def _numpy_fk(spec, q):
    N = spec.n_links
    R = [None] * N
    p = np.zeros((N, 3))
    for i in range(N):
        qr = spec.rest_quat[i].astype(np.float64)
        Q = Rotation.from_quat([qr[1], qr[2], qr[3], qr[0]])
        rel = Q * Rotation.from_euler("XY", [q[2 * i], q[2 * i + 1]])  # intrinsic x then y
        pa = spec.parent[i]
        if pa < 0:
            R[i] = rel
        else:
            R[i] = R[pa] * rel
            p[i] = p[pa] + R[pa].apply([0, 0, float(spec.length[pa])])
    return np.stack([r.as_matrix() for r in R]), p


def test_fk_matches_scipy_rotations():
    rng = np.random.default_rng(5)
    spec = stochastic_world(rng, 40, 60, 4, depth_choices=(4,))
    w = OracleWorld(spec, Params())
    q = rng.uniform(-0.6, 0.6, size=2 * spec.n_links)
    w.set_state(q=q)
    R, p, a1, a2 = w.fk()
    R2, p2 = _numpy_fk(spec, q)
    assert np.abs(R - R2).max() < 1e-12
    assert np.abs(p - p2).max() < 1e-12
    # rest pose reproduces the skeleton: Eq. 3 -> tips chain up
    w.set_state(q=np.zeros_like(q))
    R0, p0, _, _ = w.fk()
    for i in range(1, spec.n_links):
        pa = spec.parent[i]
        assert np.allclose(p0[i], p0[pa] + R0[pa] @ [0, 0, spec.length[pa]], atol=1e-13)


# ---------------------------------------------------------------- P2 mass matrix
def test_mass_matrix_single_link_closed_form():
    L, d, rho = 1.0, 0.05, 800.0
    spec = chain_spec(1, L, d, density=rho)
    w = OracleWorld(spec, Params())
    L, d = float(spec.length[0]), float(spec.diameter[0])          # the fp32 inputs both sides receive
    m = rho * math.pi * (d / 2) ** 2 * L
    J = m * L * L / 3 + m * (d / 2) ** 2 / 4
    Izz = m * (d / 2) ** 2 / 2
    assert abs(m - 1.5708) < 1e-4 and abs(J - 0.5238) < 1e-4   # SURVEY.md Appendix A values
    for th1, th2 in [(0.0, 0.0), (0.3, 0.0), (0.0, 0.7), (-0.4, 1.1)]:
        w.set_state(q=[th1, th2])
        M = w.mass_matrix()
        c, s = math.cos(th2), math.sin(th2)
        assert np.allclose(M, np.diag([J * c * c + Izz * s * s, J]), rtol=1e-12, atol=1e-15)


def test_mass_matrix_planar_double_pendulum():
    # two rods hinged about parallel x axes: textbook double pendulum (distributed mass)
    L, d, rho = 1.0, 0.04, 700.0
    spec = chain_spec(2, L, d, density=rho)
    w = OracleWorld(spec, Params())
    l = float(spec.length[0])
    r = float(spec.diameter[0]) / 2
    m = rho * math.pi * r * r * l
    Ij = m * l * l / 3 + m * r * r / 4       # rod about its own joint
    lc = l / 2
    for phi2 in (0.0, 0.5, -1.2):
        w.set_state(q=[0.2, 0.0, phi2, 0.0])
        M = w.mass_matrix()
        M11 = Ij + Ij + m * l * l + 2 * m * l * lc * math.cos(phi2)
        M12 = Ij + m * l * lc * math.cos(phi2)
        assert abs(M[0, 0] - M11) < 1e-12 and abs(M[0, 2] - M12) < 1e-12 and abs(M[2, 2] - Ij) < 1e-12


def test_mass_matrix_equals_kinetic_energy_from_fk_differences():
    """1/2 qd^T M qd = sum 1/2 m |v_cm|^2 + 1/2 w^T I w with v_cm and w obtained by central
    differences of the (separately pinned) FK output: ties RNEA columns to sum J^T I J."""
    rng = np.random.default_rng(11)
    spec = stochastic_world(rng, 20, 30, 2, depth_choices=(3, 4))
    w = OracleWorld(spec, Params())
    N = spec.n_links
    q = rng.uniform(-0.5, 0.5, size=2 * N)
    w.set_state(q=q)
    M = w.mass_matrix()
    assert np.abs(M - M.T).max() < 1e-12 * np.abs(M).max()
    assert np.linalg.eigvalsh(M).min() > 0
    dv = w.derived()
    L = spec.length.astype(np.float64)
    for trial in range(3):
        qd = rng.normal(size=2 * N)
        eps = 1e-6
        Rp, pp = _numpy_fk(spec, q + eps * qd)
        Rm, pm = _numpy_fk(spec, q - eps * qd)
        R0, _ = _numpy_fk(spec, q)
        T = 0.0
        for i in range(N):
            cp = pp[i] + Rp[i] @ [0, 0, L[i] / 2]
            cm_ = pm[i] + Rm[i] @ [0, 0, L[i] / 2]
            v = (cp - cm_) / (2 * eps)
            Wm = (Rp[i] - Rm[i]) / (2 * eps) @ R0[i].T          # [w]x
            wv = np.array([Wm[2, 1], Wm[0, 2], Wm[1, 0]])
            wl = R0[i].T @ wv
            T += 0.5 * dv["m"][i] * v @ v + 0.5 * (dv["Ixx"][i] * (wl[0] ** 2 + wl[1] ** 2) + dv["Izz"][i] * wl[2] ** 2)
        assert abs(0.5 * qd @ M @ qd - T) < 1e-7 * T


# ---------------------------------------------------------------- P3 gravity
def test_gravity_torque_horizontal_rod():
    L, d, rho = 1.0, 0.05, 800.0
    spec = chain_spec(1, L, d, root_quat=quat_axis("x", -90.0), density=rho)   # +z of the link -> world +y
    w = OracleWorld(spec, Params())
    L, d = float(spec.length[0]), float(spec.diameter[0])
    m = rho * math.pi * (d / 2) ** 2 * L
    tau = w.rnea()
    assert abs(abs(tau[0]) - m * G * L / 2) < 1e-12 * m * G * L and abs(tau[1]) < 1e-12
    assert abs(m * G * L / 2 - 7.7048) < 1e-4


# ---------------------------------------------------------------- P4 cantilever
@pytest.mark.parametrize("n", [1, 2, 4, 8, 16, 32])
def test_cantilever_tip_deflection(n):
    """n-link horizontal cantilever, tip load P, no gravity, small load:
    delta_n = (P L^3 / EI) (n+1)(2n+1)/(6 n^2)  ->  P L^3/(3EI) as n grows (north_star)."""
    L, d, E, Pload = 1.0, 0.05, 8e9, 0.1
    spec = chain_spec(n, L, d, root_quat=quat_axis("x", -90.0), E=E)
    par = Params(h=50.0, gravity=(0.0, 0.0, 0.0), c_d=0.0, qd_max=0.0)
    w = OracleWorld(spec, par)
    w.apply_wrench(n - 1, (0, 0, float(spec.length[-1])), (0, 0, -Pload))
    _, p0, _, _ = w.fk()
    R0, _, _, _ = w.fk()
    tip0 = p0[-1] + R0[-1] @ [0, 0, float(spec.length[-1])]
    w.step(6)          # huge h: each step is a Newton step of the static problem
    R, p, _, _ = w.fk()
    tip = p[-1] + R[-1] @ [0, 0, float(spec.length[-1])]
    EI = E * math.pi * float(spec.diameter[0]) ** 4 / 64
    Ltot = float(spec.length.astype(np.float64).sum())
    delta = Pload * Ltot ** 3 / EI * (n + 1) * (2 * n + 1) / (6 * n * n)
    got = -(tip - tip0)[2]
    assert abs(got / delta - 1) < 2e-6
    ratio = got / (Pload * Ltot ** 3 / (3 * EI))
    assert abs(ratio - (1 + 1.5 / n + 0.5 / n ** 2)) < 1e-5


# ---------------------------------------------------------------- P5 linear dynamics
def test_single_dof_step_map_closed_form():
    L, d, rho, E = 0.6, 0.02, 800.0, 1e8
    spec = chain_spec(1, L, d, density=rho, E=E)
    h, c_d = 2e-3, 0.05
    par = Params(h=h, gravity=(0, 0, 0), c_d=c_d, qd_max=0.0)
    w = OracleWorld(spec, par)
    hh, cd = float(np.float32(h)), float(np.float32(c_d))
    r = float(spec.diameter[0]) / 2
    Lf = float(spec.length[0])
    m = rho * math.pi * r * r * Lf
    J = m * Lf * Lf / 3 + m * r * r / 4
    K = E * math.pi * (2 * r) ** 4 / (64 * Lf)
    D = cd * K
    q, v = 0.01, -0.3
    w.set_state(q=[0.0, q], qd=[0.0, v])
    for _ in range(50):
        v = (J * v - hh * K * q) / (J + hh * D + hh * hh * K)
        q = q + hh * v
        w.step(1)
        s = w.get_state()
        assert abs(s["q"][1] - q) < 1e-13 and abs(s["qd"][1] - v) < 1e-11
        assert s["q"][0] == 0.0 and s["qd"][0] == 0.0


def test_small_oscillation_frequencies_match_generalized_eigenvalues():
    """log-eigenvalues of the linearised step map / h -> sqrt(eig(K, M)) for D = 0, h -> 0 (north_star)."""
    rng = np.random.default_rng(3)
    spec = stochastic_world(rng, 6, 8, 0, depth_choices=(2,))
    spec = dataclasses.replace(spec, E=2e6)
    h = 1e-4
    par = Params(h=h, gravity=(0, 0, 0), c_d=0.0, qd_max=0.0)
    w = OracleWorld(spec, par)
    n = 2 * spec.n_links
    M = w.mass_matrix()
    Kd = np.repeat(w.derived()["K"], 2)
    lam = scipy.linalg.eigh(np.diag(Kd), M, eigvals_only=True)
    omega_ref = np.sqrt(lam)
    # linearise the step map by central differences about rest
    eps = 1e-7
    S = np.zeros((2 * n, 2 * n))
    for j in range(2 * n):
        cols = []
        for sgn in (+1, -1):
            x = np.zeros(2 * n)
            x[j] = sgn * eps
            w.set_state(q=x[:n], qd=x[n:])
            w.step(1)
            s = w.get_state()
            cols.append(np.concatenate([s["q"], s["qd"]]))
        S[:, j] = (cols[0] - cols[1]) / (2 * eps)
    ev = np.linalg.eigvals(S)
    assert np.abs(ev).max() < 1.0 + 1e-9          # never unstable
    omega = np.sort(np.abs(np.log(ev).imag) / float(np.float32(h)))
    omega = omega[::2]                             # conjugate pairs
    assert np.allclose(omega, np.sort(omega_ref), rtol=2e-3)


# ---------------------------------------------------------------- P16 Lagrangian brute force
def test_single_link_two_dof_against_hand_derived_lagrangian():
    """Universal joint + symmetric rod: T = 1/2 (J c2^2 + Izz s2^2) th1'^2 + 1/2 J th2'^2,
    V = -m (L/2) g . R e_z with R e_z = (s2, -s1 c2, c1 c2); same linearly implicit scheme."""
    L, d, rho, E = 0.8, 0.03, 800.0, 3e5
    spec = chain_spec(1, L, d, density=rho, E=E, root_quat=quat_axis("y", 40.0))
    h, c_d = 1e-3, 0.02
    gvec = (0.3, -0.2, -9.81)
    par = Params(h=h, gravity=gvec, c_d=c_d, qd_max=0.0)
    w = OracleWorld(spec, par)
    hh, cd = float(np.float32(h)), float(np.float32(c_d))
    r = float(spec.diameter[0]) / 2
    Lf = float(spec.length[0])
    m = rho * math.pi * r * r * Lf
    J = m * Lf * Lf / 3 + m * r * r / 4
    Izz = m * r * r / 2
    K = E * math.pi * (2 * r) ** 4 / (64 * Lf)
    D = cd * K
    qr = spec.rest_quat[0].astype(np.float64)
    Q = Rotation.from_quat([qr[1], qr[2], qr[3], qr[0]]).as_matrix()
    gl = Q.T @ np.array([float(np.float32(x)) for x in gvec])      # gravity in the joint's rest frame
    q = np.array([0.3, -0.5])
    v = np.array([1.0, 2.0])
    w.set_state(q=q, qd=v)
    for _ in range(300):
        s1, c1, s2, c2 = math.sin(q[0]), math.cos(q[0]), math.sin(q[1]), math.cos(q[1])
        M11 = J * c2 * c2 + Izz * s2 * s2
        dM11 = 2 * (Izz - J) * s2 * c2
        cor = np.array([dM11 * v[0] * v[1], -0.5 * dM11 * v[0] ** 2])
        dV = -m * Lf / 2 * np.array([gl @ [0, -c1 * c2, -s1 * c2], gl @ [c2, s1 * s2, -c1 * s2]])
        A = np.diag([M11, J]) + np.eye(2) * (hh * D + hh * hh * K)
        b = hh * (-cor - dV - K * q - (D + hh * K) * v)
        v = v + np.linalg.solve(A, b)
        q = q + hh * v
        w.step(1)
    s = w.get_state()
    assert np.abs(s["q"] - q).max() < 1e-10 and np.abs(s["qd"] - v).max() < 1e-9


# ---------------------------------------------------------------- P6 / P7 energy, order
def _soft_tree():
    rng = np.random.default_rng(21)
    spec = stochastic_world(rng, 14, 18, 0, depth_choices=(3,))
    return dataclasses.replace(spec, E=3e6)


def _energy_run(h, t_end=0.5):
    spec = _soft_tree()
    w = OracleWorld(spec, Params(h=h, c_d=0.0, qd_max=0.0))
    T0, V0 = w.energy()
    Es = [T0 + V0]
    Tmax = 0.0
    for _ in range(int(round(t_end / h))):
        w.step(1)
        T, V = w.energy()
        Es.append(T + V)
        Tmax = max(Tmax, T)
    return np.array(Es), Tmax, w.get_state()


def test_energy_drift_is_first_order_and_never_grows():
    drift = []
    for h in (1e-3, 5e-4, 2.5e-4):
        Es, Tmax, _ = _energy_run(h)
        assert Tmax > 0
        rel = (Es - Es[0]) / Tmax
        assert rel.max() < 1e-9             # never gains energy (implicit spring, D = 0)
        drift.append(rel[-1])
    assert drift[0] < 0 and abs(drift[0]) < 0.05          # small
    assert 1.6 < drift[0] / drift[1] < 2.4 and 1.6 < drift[1] / drift[2] < 2.4


def test_first_order_convergence_in_h():
    _, _, ref = _energy_run(2.5e-5, t_end=0.1)
    errs = []
    for h in (4e-4, 2e-4, 1e-4):
        _, _, s = _energy_run(h, t_end=0.1)
        errs.append(np.linalg.norm(s["q"] - ref["q"]))
    assert 1.6 < errs[0] / errs[1] < 2.5 and 1.6 < errs[1] / errs[2] < 2.7


# ---------------------------------------------------------------- P8 rupture
def test_rupture_fires_exactly_at_the_closed_form_moment():
    L, d = 0.5, 0.02
    big = np.full((1, 2), 1e9, dtype=np.float32)       # armature pins the joint in place
    spec = chain_spec(1, L, d, armature=big)
    Mmax = 60e6 * math.pi * float(spec.diameter[0]) ** 3 / 32
    K = 8e9 * math.pi * float(spec.diameter[0]) ** 4 / (64 * float(spec.length[0]))
    for nr in (1, 3, 5):
        for factor, fires in ((1 + 1e-3, True), (1 - 1e-3, False)):
            w = OracleWorld(spec, Params(gravity=(0, 0, 0), rupture_frames=nr))
            th = factor * Mmax / K
            w.set_state(q=[0.6 * th, 0.8 * th])
            w.step(nr - 1) if nr > 1 else None
            assert w.events() == []
            w.step(4)
            ev = w.events()
            if fires:
                assert len(ev) == 1 and ev[0][1] == nr - 1 and ev[0][2] == 0 and ev[0][3] == 0
                assert abs(ev[0][4] / (factor * Mmax) - 1) < 1e-6 and abs(ev[0][5] / Mmax - 1) < 1e-12
                assert w.get_state()["ruptured"][0] == 1
            else:
                assert ev == [] and w.get_state()["ruptured"][0] == 0


def test_rupture_under_quasi_static_ramp():
    """One horizontal link, N_r = 1, slow tip-load ramp: at the first event P L cos(theta) is within the
    damper lag (c_d dP/dt L) of M_max = MOR pi d^3/32."""
    L, d, E, MOR = 0.4, 0.01, 8e9, 60e6
    spec = chain_spec(1, L, d, root_quat=quat_axis("x", -90.0), E=E, MOR=MOR)
    h, c_d, nsteps = 2e-3, 0.05, 4000
    Mmax = MOR * math.pi * float(spec.diameter[0]) ** 3 / 32
    Lf = float(spec.length[0])
    Pmax = 1.5 * Mmax / Lf
    w = OracleWorld(spec, Params(h=h, c_d=c_d, gravity=(0, 0, 0), rupture_frames=1, qd_max=0.0))
    ev = []
    for s in range(nsteps):
        w.apply_wrench(0, (0, 0, Lf), (0, 0, -Pmax * (s + 1) / nsteps))
        w.step(1)
        ev = w.events()
        if ev:
            break
    assert ev and ev[0][2] == 0
    s = ev[0][1]
    th = np.linalg.norm(w.get_state()["q"])
    P = Pmax * (s + 1) / nsteps
    lag = c_d * (Pmax / (nsteps * h)) * Lf
    assert abs(P * Lf * math.cos(th) - Mmax) < lag + 2 * Pmax / nsteps * Lf + 1e-3 * Mmax
    assert ev[0][4] > ev[0][5] and ev[0][4] / ev[0][5] < 1.001


def test_ruptured_joint_is_a_free_hinge():
    L, d, rho = 0.5, 0.02, 800.0
    spec = chain_spec(1, L, d, root_quat=quat_axis("x", -90.0), density=rho)
    h = 1e-3
    w = OracleWorld(spec, Params(h=h, qd_max=0.0))
    w.set_state(ruptured=[1])
    w.step(1)
    r = float(spec.diameter[0]) / 2
    Lf = float(spec.length[0])
    m = rho * math.pi * r * r * Lf
    J = m * Lf * Lf / 3 + m * r * r / 4
    qd = w.get_state()["qd"]
    assert abs(abs(qd[0]) - float(np.float32(h)) * (m * G * Lf / 2) / J) < 1e-12 and abs(qd[1]) < 1e-14


# ---------------------------------------------------------------- P9 / P10 / P11 apples
def test_config1_events_as_written_and_1b():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "config1_events.txt")) if l.strip() and l[0] != "#"]
    spec = binary_tree_config1()
    for variant, fmax in (("1", 400.0), ("1b", 5000.0)):
        for implicit in (1, 0):                                   # P11: explicit and implicit tether agree
            P = dataclasses.replace(config_params(1), tether_implicit=implicit)
            w = OracleWorld(spec, P)
            for s in range(500):
                for (_, body, pt, f) in config1_loads(spec, s, 500, 30.0, fmax):
                    w.apply_wrench(body, pt, f)
                w.step(1)
            ev = w.events()
            exp = [r for r in rows if r[0] == variant]
            assert len(ev) == len(exp), (variant, implicit, ev)
            for e, r in zip(ev, exp):
                step, kind, index, value, thr = int(r[1]), int(r[2]), int(r[3]), float(r[4]), float(r[5])
                assert e[2] == kind and e[3] == index
                if kind == 1:
                    assert e[1] == step and abs(e[4] - value) < 1e-5 and abs(e[5] - thr) < 1e-6
                else:
                    assert abs(e[1] - step) <= 2 and 1.0 < e[4] / e[5] < 1.01 and abs(e[5] - thr) < 0.1
            assert w.get_state()["status"] == 0


def test_detach_by_stem_tension_path():
    """Slow vertical pull on a hanging apple: |f_s| = P + m g quasi-statically, path B fires when it has
    exceeded kappa f_detach for N_B steps (reading A14)."""
    mA, k, fdet = 0.2, 2e3, 20.0
    spec = chain_spec(1, 0.5, 0.08, apples=[(0, (0, 0, 0.5), mA, k, fdet)])
    P = Params(detach_frames_pull=10 ** 6, detach_frames_tension=10, zeta_s=1.0)
    w = OracleWorld(spec, P)
    nsteps = 6000
    Pmax = 30.0
    fired = None
    for s in range(nsteps):
        w.apply_wrench(1, (0, 0, 0), (0, 0, -Pmax * (s + 1) / nsteps))
        w.step(1)
        ev = w.events()
        if ev:
            fired = ev[0]
            break
    assert fired is not None and fired[2] == 1 and fired[3] == 0
    thr = float(np.float32(1.1)) * fdet
    assert abs(fired[5] - thr) < 1e-9
    s10 = fired[1] - 9                                    # first step of the 10-step window
    Pq = Pmax * (s10 + 1) / nsteps
    # quasi-static balance on the apple: f_s = P + m g - c_s |v|, with v = (dP/dt)/k_s the ramp-following speed
    c_s = 2.0 * 1.0 * math.sqrt(k * mA)
    lag = c_s * (Pmax / (nsteps * 2e-3)) / k
    assert abs((Pq + mA * G - lag) - thr) < 2 * Pmax / nsteps


def test_apple_rest_sag_zero_reaction_and_identical_tree():
    spec = binary_tree_config1()
    P = config_params(1)
    w = OracleWorld(spec, P)
    s0 = w.get_state()
    R, p, _, _ = w.fk()
    for a in range(spec.n_apples):
        b = spec.apple_link[a]
        xh = p[b] + R[b] @ spec.apple_offset[a].astype(np.float64)
        sag = xh - s0["apple_x"][a]
        assert np.allclose(sag, [0, 0, float(spec.apple_mass[a]) * G / float(spec.apple_k[a])], atol=1e-9)
    w0 = OracleWorld(strip_apples(spec), P)
    A1, b1 = w.system()
    A0, b0 = w0.system()
    assert np.abs(b1 - b0).max() < 1e-9 * np.abs(b0).max()      # zero reaction at rest
    w.step(100)
    w0.step(100)
    assert np.abs(w.get_state()["q"] - w0.get_state()["q"]).max() < 5e-6
    assert w.events() == []


def test_virtual_mass_identity():
    """h^2 k_s J^T J (A15) equals the mass-matrix increment of a point mass h^2 k_s at the attach point:
    checked with a heavy, short, thin extra link standing in for the point mass."""
    spec = binary_tree_config1()
    P = config_params(1)
    w = OracleWorld(spec, P)
    rng = np.random.default_rng(2)
    q = rng.uniform(-0.2, 0.2, size=2 * spec.n_links)
    w.set_state(q=q)
    A1, _ = w.system()
    w0 = OracleWorld(strip_apples(spec), P)
    w0.set_state(q=q)
    A0, _ = w0.system()
    dA = A1 - A0
    R, p, a1, a2 = w.fk()
    hh = float(np.float32(P.h))
    ref = np.zeros_like(dA)
    for a in range(spec.n_apples):
        b = int(spec.apple_link[a])
        xh = p[b] + R[b] @ spec.apple_offset[a].astype(np.float64)
        J = np.zeros((3, 2 * spec.n_links))
        j = b
        while j >= 0:
            J[:, 2 * j] = np.cross(a1[j], xh - p[j])
            J[:, 2 * j + 1] = np.cross(a2[j], xh - p[j])
            j = int(spec.parent[j])
        ref += hh * hh * float(spec.apple_k[a]) * J.T @ J
    assert np.abs(dA - ref).max() < 1e-12 * np.abs(ref).max()
    # and J is the true Jacobian of the hang point (finite differences of FK)
    eps = 1e-6
    b = int(spec.apple_link[0])
    o = spec.apple_offset[0].astype(np.float64)
    for j in (0, 1, 2 * b, 2 * b + 1):
        dq = np.zeros_like(q)
        dq[j] = eps
        Rp, pp = _numpy_fk(spec, q + dq)
        Rm, pm = _numpy_fk(spec, q - dq)
        col = ((pp[b] + Rp[b] @ o) - (pm[b] + Rm[b] @ o)) / (2 * eps)
        jj = b
        Jc = np.zeros(3)
        xh = p[b] + R[b] @ o
        while jj >= 0:
            if 2 * jj == j:
                Jc = np.cross(a1[jj], xh - p[jj])
            if 2 * jj + 1 == j:
                Jc = np.cross(a2[jj], xh - p[jj])
            jj = int(spec.parent[jj])
        assert np.abs(col - Jc).max() < 1e-8


# ---------------------------------------------------------------- P13 PCG vs Cholesky
def test_fp64_pcg_equals_cholesky():
    rng = np.random.default_rng(8)
    spec = stochastic_world(rng, 60, 80, 6, depth_choices=(4, 5))
    P = config_params(2)
    a = OracleWorld(spec, P, solver=0)
    b = OracleWorld(spec, P, solver=1)
    b.set_solver(1, 1e-13, 5000)
    for w in (a, b):
        w.randomize(99)
        w.apply_wrench(10, (0, 0, 0.01), (3.0, -2.0, 1.0))
    a.step(20)
    b.step(20)
    sa, sb = a.get_state(), b.get_state()
    assert np.abs(sa["q"] - sb["q"]).max() < 1e-10 and np.abs(sa["qd"] - sb["qd"]).max() < 1e-8
    assert 0 < sb["last_iters"] < 200


# ---------------------------------------------------------------- P14 symmetry
def test_config1_c2_symmetry_under_gravity():
    spec = binary_tree_config1()
    w = OracleWorld(spec, config_params(1))
    w.step(100)
    q = w.get_state()["q"].reshape(-1, 2)
    nrm = np.linalg.norm(q, axis=1)
    for i, j in [(1, 2), (3, 5), (4, 6), (7, 11), (15, 23), (16, 24), (19, 27)]:
        assert nrm[i] > 0 and abs(nrm[i] - nrm[j]) < 1e-9 * nrm[i]


# ---------------------------------------------------------------- P15 restart after rupture
def test_state_round_trip_reproduces_the_run_after_a_rupture():
    spec = binary_tree_config1()
    P = config_params(1)
    a = OracleWorld(spec, P)
    for s in range(460):
        for (_, body, pt, f) in config1_loads(spec, s, 500, 30.0, 5000.0):
            a.apply_wrench(body, pt, f)
        a.step(1)
    st = a.get_state()
    assert st["ruptured"][4] == 1 and st["attached"][0] == 0
    b = OracleWorld(spec, P)
    b.set_state(st["q"], st["qd"], st["apple_x"], st["apple_v"], st["ruptured"], st["attached"])
    for w in (a, b):
        for (_, body, pt, f) in config1_loads(spec, 460, 500, 30.0, 5000.0):
            w.apply_wrench(body, pt, f)
        w.step(20)
    sa, sb = a.get_state(), b.get_state()
    assert np.abs(sa["q"] - sb["q"]).max() < 1e-12 and np.abs(sa["apple_x"] - sb["apple_x"]).max() < 1e-12
    # forces on a snapped sub-tree are disabled (reading A10): the load on link 4 no longer matters
    c = OracleWorld(spec, P)
    c.set_state(st["q"], st["qd"], st["apple_x"], st["apple_v"], st["ruptured"], st["attached"])
    c.apply_wrench(spec.n_links + 0, (0, 0, 0), config1_loads(spec, 460, 500, 30.0, 5000.0)[0][3])
    c.step(20)
    assert np.abs(c.get_state()["q"] - sb["q"]).max() < 1e-12


# ---------------------------------------------------------------- A32: mass-proportional damping
def test_mass_damping_single_dof_step_map_closed_form():
    """(J (1 + h a) + h D + h^2 K) dv = h [-K q - (D + h K) v - a J v]: the 1-DoF step map with F = -c_v m v,
    tau = -c_omega I omega (c_v = c_omega = a) taken implicitly, written out by hand."""
    L, d, rho, E = 0.6, 0.02, 800.0, 1e8
    spec = chain_spec(1, L, d, density=rho, E=E)
    h, c_d, a = 2e-3, 0.05, 3.0
    w = OracleWorld(spec, Params(h=h, gravity=(0, 0, 0), c_d=c_d, qd_max=0.0, mass_damping=a))
    hh, cd = float(np.float32(h)), float(np.float32(c_d))
    r, Lf = float(spec.diameter[0]) / 2, float(spec.length[0])
    m = rho * math.pi * r * r * Lf
    J = m * Lf * Lf / 3 + m * r * r / 4
    K = E * math.pi * (2 * r) ** 4 / (64 * Lf)
    D = cd * K
    q, v = 0.01, -0.3
    w.set_state(q=[0.0, q], qd=[0.0, v])
    for _ in range(50):
        v = v + hh * (-K * q - (D + hh * K) * v - a * J * v) / (J * (1 + hh * a) + hh * D + hh * hh * K)
        q = q + hh * v
        w.step(1)
        s = w.get_state()
        assert abs(s["q"][1] - q) < 1e-13 and abs(s["qd"][1] - v) < 1e-11


def test_mass_damping_free_hinge_decays_geometrically_and_dissipates_2aT():
    """A ruptured (free) hinge without gravity: v_n = v_0 / (1 + h a)^n exactly; on a tree the kinetic energy
    falls at the rate -2 a T (power of F = -a m v, tau = -a I omega summed over the links), to first order in h."""
    spec = chain_spec(1, 0.5, 0.02)
    h, a = 1e-3, 2.0
    w = OracleWorld(spec, Params(h=h, gravity=(0, 0, 0), qd_max=0.0, mass_damping=a))
    w.set_state(qd=[0.0, 1.5], ruptured=[1])
    hh = float(np.float32(h))
    for n in range(1, 40):
        w.step(1)
        assert abs(w.get_state()["qd"][1] - 1.5 / (1 + hh * a) ** n) < 1e-13
    # energy rate on a soft, undamped, gravity-free tree
    rng = np.random.default_rng(5)
    tree = strip_apples(stochastic_world(rng, 20, 30, 0, depth_choices=(3,)))
    tree = dataclasses.replace(tree, E=1e-3)               # springs negligible: kinetic energy only
    par = Params(h=1e-4, gravity=(0, 0, 0), c_d=0.0, qd_max=0.0, mass_damping=a)
    w = OracleWorld(tree, par)
    qd0 = 0.3 * rng.standard_normal(2 * tree.n_links)
    w.set_state(qd=qd0)
    T0, _ = w.energy()
    w.step(100)
    T1, _ = w.energy()
    t = 100 * float(np.float32(1e-4))
    assert abs(math.log(T1 / T0) / t + 2 * a) < 2e-2 * 2 * a


def test_mass_damping_on_a_detached_apple():
    """v <- v + h (g - a v): the detached apple is a point body with F = -c_v m v (explicit)."""
    spec = chain_spec(1, 0.5, 0.02, apples=[(0, (0, 0, 0.5), 0.2, 2e3, 20.0)])
    h, a = 2e-3, 1.5
    w = OracleWorld(spec, Params(h=h, qd_max=0.0, mass_damping=a))
    w.set_state(attached=[0], apple_v=[[0.4, 0.0, -0.2]])
    hh = float(np.float32(h))
    v = np.array([0.4, 0.0, -0.2])
    for _ in range(20):
        v = v + hh * (np.array([0.0, 0.0, -G]) - a * v)
        w.step(1)
        assert np.abs(w.get_state()["apple_v"][0] - v).max() < 1e-13


# ---------------------------------------------------------------- Eq. 1: ternary L-system workload (8(f) item 4)
def test_ternary_lsystem_body_count_and_oracle_rest():
    """after n derivations the body count is 1 + 2 (3^n - 1); every apex carries three branches and
    one straight continuation; the tree is at rest in the oracle (apples hang m g / k_s below their tips)."""
    from workloads import ternary_lsystem_world
    for n in (1, 2, 3, 4):
        w = ternary_lsystem_world(n, 30)
        assert w.n_links == 1 + 2 * (3 ** n - 1)
        kids = np.bincount(w.parent[1:], minlength=w.n_links)
        assert sorted(set(kids.tolist())) == [0, 1, 3] and (kids == 0).sum() == 3 ** n
        assert np.all(w.parent[1:] < np.arange(1, w.n_links))
    w = ternary_lsystem_world(3, 9)
    ow = OracleWorld(w, Params(h=1e-3, gravity=(0, 0, 0)))
    ow.step(5)
    s = ow.get_state()
    assert np.abs(s["q"]).max() < 1e-12 and np.abs(s["qd"]).max() < 1e-10


# ---------------------------------------------------------------- Eq. 7 clamp, implicit-tether term, speed clamp, wrench slots
def _fd_jacobian(spec, q, link, offset, eps=1e-6):
    """3 x n Jacobian of the world position of a link-fixed point, by central differences of the scipy FK."""
    n = 2 * spec.n_links
    J = np.zeros((3, n))
    o = np.asarray(offset, dtype=np.float64)
    for j in range(n):
        dq = np.zeros(n)
        dq[j] = eps
        Rp, pp = _numpy_fk(spec, q + dq)
        Rm, pm = _numpy_fk(spec, q - dq)
        J[:, j] = ((pp[link] + Rp[link] @ o) - (pm[link] + Rm[link] @ o)) / (2 * eps)
    return J


def _tether_rhs(spec, P, q, qd, apple_x):
    """b(tree with the apple) - b(the same tree without it): the generalized force of the tether reaction times h."""
    w1 = OracleWorld(spec, P)
    w1.set_state(q=q, qd=qd, apple_x=apple_x)
    w0 = OracleWorld(strip_apples(spec), P)
    w0.set_state(q=q, qd=qd)
    return w1.system()[1] - w0.system()[1]


def test_tether_reaction_norm_clamp_at_react_max():
    """Eq. 7 + PAPER.md:161 (A13): f_react = k_s (x_a - x_hang) + m g zhat, clamped in NORM to react_max = 40 N.
    b_with - b_without = h J^T f_react with J the finite-difference Jacobian of the hang point.
    (Perturbations this fails on: no clamp; a component-wise clamp; clamping before adding m g.)"""
    mA, ks, off = 0.2, 2e3, (0.01, -0.02, 0.13)
    spec = chain_spec(3, 0.9, 0.03, root_quat=quat_axis("y", 70.0), apples=[(2, off, mA, ks, 20.0)])
    P = Params(h=2e-3, react_max=40.0)
    h = float(np.float32(P.h))
    rng = np.random.default_rng(12)
    q = rng.uniform(-0.15, 0.15, size=6)
    R, p = _numpy_fk(spec, q)
    xh = p[2] + R[2] @ np.array(off, dtype=np.float64)
    J = _fd_jacobian(spec, q, 2, off)
    d = np.array([0.6, -0.3, 0.74])
    d /= np.linalg.norm(d)
    for stretch, clamped in ((0.004, False), (0.0185, False), (0.0215, True), (0.05, True)):
        x_a = xh + stretch * d
        f = ks * (x_a - xh) + np.array([0.0, 0.0, mA * G])
        assert (np.linalg.norm(f) > 40.0) == clamped
        if clamped:
            f = f * (40.0 / np.linalg.norm(f))
        db = _tether_rhs(spec, P, q, np.zeros(6), [x_a])
        assert np.abs(db - h * J.T @ f).max() < 2e-7 * np.abs(db).max(), (stretch, db, h * J.T @ f)


def test_implicit_tether_term_eta_h_v_hang():
    """A15: the reaction is taken at the hang point advanced by eta h v_hang, v_hang = J qd (point_velocity).
    The tether part of b changes with qd by exactly -h^2 k_s J^T J qd in implicit mode and by 0 with
    tether_implicit = 0.  (Perturbations this fails on: the sign of the term; v_hang of the link origin instead of
    the hang point; a missing ancestor in the velocity sum.)"""
    mA, ks, off = 0.2, 2e3, (0.015, 0.01, 0.11)
    spec = chain_spec(3, 0.9, 0.03, root_quat=quat_axis("y", 70.0), apples=[(2, off, mA, ks, 20.0)])
    rng = np.random.default_rng(13)
    q = rng.uniform(-0.15, 0.15, size=6)
    qd = rng.uniform(-0.8, 0.8, size=6)
    R, p = _numpy_fk(spec, q)
    xh = p[2] + R[2] @ np.array(off, dtype=np.float64)
    x_a = xh + np.array([0.001, -0.002, -0.0015])            # 5 N of stretch: far below the clamp
    J = _fd_jacobian(spec, q, 2, off)
    for eta in (1, 0):
        P = Params(h=2e-3, tether_implicit=eta)
        h = float(np.float32(P.h))
        diff = _tether_rhs(spec, P, q, qd, [x_a]) - _tether_rhs(spec, P, q, np.zeros(6), [x_a])
        expect = -eta * h * h * ks * (J.T @ (J @ qd))
        scale = h * h * ks * np.abs(J.T @ (J @ qd)).max()
        assert np.abs(diff - expect).max() < 1e-6 * scale, (eta, diff, expect)


def test_joint_speed_clamp_componentwise_and_q_uses_the_clamped_speed():
    """A16: qd+ = clamp(qd + dqd, +-qd_max) component-wise, q+ = q + h qd+ with the clamped value.
    The unclamped update comes from a twin world with the clamp disabled.  (Perturbations this fails on: no clamp;
    a norm clamp over the two DoF of a joint; q advanced with the unclamped speed.)"""
    spec = chain_spec(2, 0.6, 0.004, root_quat=quat_axis("x", -90.0), E=2e8)
    q0 = np.array([0.02, -0.01, 0.03, 0.015])
    qd0 = np.array([56.0, -12.0, -61.0, 49.0])
    free = OracleWorld(spec, Params(h=2e-3, qd_max=0.0))
    free.set_state(q=q0, qd=qd0)
    free.step(1)
    v = free.get_state()["qd"]
    assert (np.abs(v) > 50.0).sum() >= 2 and (np.abs(v) < 50.0).sum() >= 1     # the case exercises both branches
    w = OracleWorld(spec, Params(h=2e-3, qd_max=50.0))
    w.set_state(q=q0, qd=qd0)
    w.step(1)
    s = w.get_state()
    vc = np.clip(v, -50.0, 50.0)
    assert np.abs(s["qd"] - vc).max() == 0.0
    assert np.abs(s["q"] - (q0 + float(np.float32(2e-3)) * vc)).max() < 1e-15


def test_wrench_slot_semantics():
    """a wrench persists, a second one on the same body REPLACES it, a zero force frees the slot,
    distinct bodies superpose, a ninth distinct body is refused (rc -2) until a slot is freed.  Checked on the
    right-hand side b, which is affine in the applied forces."""
    spec = binary_tree_config1()
    P = config_params(1)
    w = OracleWorld(spec, P)
    rng = np.random.default_rng(14)
    q = rng.uniform(-0.05, 0.05, size=2 * spec.n_links)

    def rhs(loads):
        x = OracleWorld(spec, P)
        x.set_state(q=q)
        for (body, pt, f) in loads:
            x.apply_wrench(body, pt, f)
        return x.system()[1]
    b0 = rhs([])
    F1, F2 = (5.0, -3.0, 2.0), (-1.0, 4.0, 6.0)
    b1 = rhs([(4, (0, 0, 0.2), F1)])
    b2 = rhs([(9, (0.01, 0, 0.1), F2)])
    assert np.abs(b1 - b0).max() > 1e-6 and np.abs(b2 - b0).max() > 1e-6
    assert np.abs(rhs([(4, (0, 0, 0.2), F2), (4, (0, 0, 0.2), F1)]) - b1).max() < 1e-15        # replace, not add
    assert np.abs(rhs([(4, (0, 0, 0.2), F1), (4, (0, 0, 0), (0, 0, 0))]) - b0).max() == 0.0     # zero frees
    both = rhs([(4, (0, 0, 0.2), F1), (9, (0.01, 0, 0.1), F2)])
    assert np.abs((both - b0) - ((b1 - b0) + (b2 - b0))).max() < 1e-12 * np.abs(both).max()     # distinct bodies add
    for body in range(8):
        w.apply_wrench(body, (0, 0, 0.1), (1.0, 0, 0))
    w.apply_wrench(3, (0, 0, 0.1), (2.0, 0, 0))                  # same body: no new slot
    with pytest.raises(RuntimeError):
        w.apply_wrench(20, (0, 0, 0.1), (1.0, 0, 0))             # ninth distinct body
    w.apply_wrench(0, (0, 0, 0), (0, 0, 0))
    w.apply_wrench(20, (0, 0, 0.1), (1.0, 0, 0))                 # fits after the free
    with pytest.raises(RuntimeError):
        w.apply_wrench(spec.n_links + spec.n_apples, (0, 0, 0), (1.0, 0, 0))   # body out of range
    # a wrench on an apple is a force on the apple, not on the tree: b is unchanged, the apple accelerates
    ba = rhs([(spec.n_links + 1, (0, 0, 0), (0.0, 3.0, 0.0))])
    assert np.abs(ba - b0).max() == 0.0


# ---------------------------------------------------------------- per-world geometry randomization (8(f) item 3, A37)
def _u32_uniform(x, lo, hi):
    u = np.float32(int(x) >> 8) * np.float32(2.0 ** -24)
    return np.float32(np.float64(u) * np.float64(np.float32(hi) - np.float32(lo)) + np.float64(np.float32(lo)))


def test_geometry_randomization_zero_strength_reproduces_the_base_model():
    """the on-device build "reproduces the replicated base model exactly at zero strength"."""
    rng = np.random.default_rng(21)
    spec = stochastic_world(rng, 60, 90, 8, depth_choices=(4, 5))
    P = config_params(2)
    w = OracleWorld(spec, P, world_index=3)
    g0, A0, b0, s0 = w.geometry(), *w.system(), w.get_state()
    w.randomize_geometry(12345)
    g1, (A1, b1), s1 = w.geometry(), w.system(), w.get_state()
    for k in g0:
        assert np.array_equal(g0[k], g1[k]) if k != "Q" else np.abs(g0[k] - g1[k]).max() < 1e-15, k
    assert np.abs(A1 - A0).max() <= 1e-12 * np.abs(A0).max() and np.abs(s1["apple_x"] - s0["apple_x"]).max() < 1e-13


def test_geometry_randomization_dimensions_follow_the_draws():
    """Reading A37: L_i = (L0_i * scale) * jitter_i in fp32 (stream 3 item 1, stream 4 item i), diameters likewise;
    K, M_max, m follow Eq. 4 / Eq. 5; apple offsets scale with their link; apples hang at rest under the new tips."""
    rng = np.random.default_rng(22)
    spec = stochastic_world(rng, 40, 60, 6, depth_choices=(4,))
    w = OracleWorld(spec, config_params(2), world_index=5)
    seed = (9 << 32) | 77
    rg = dict(scale_length=(0.8, 1.25), scale_diameter=(0.7, 1.3), jitter_length=(0.9, 1.1), jitter_diameter=(0.85, 1.15))
    w.randomize_geometry(seed, **rg)
    key = [seed & 0xffffffff, seed >> 32]
    o = philox4x32_10([5, 1, 3, 0], key)
    sL, sD = _u32_uniform(o[1], *rg["scale_length"]), _u32_uniform(o[2], *rg["scale_diameter"])
    g = w.geometry()
    for i in range(spec.n_links):
        oi = philox4x32_10([5, i, 4, 0], key)
        Ln = np.float32(np.float32(spec.length[i] * sL) * _u32_uniform(oi[0], *rg["jitter_length"]))
        dn = np.float32(np.float32(spec.diameter[i] * sD) * _u32_uniform(oi[1], *rg["jitter_diameter"]))
        assert g["length"][i] == float(Ln) and g["diameter"][i] == float(dn), i
    d = w.derived()
    E, rho = float(np.float32(spec.E)), float(np.float32(spec.density))
    assert np.allclose(d["K"], E * math.pi * g["diameter"] ** 4 / (64 * g["length"]), rtol=1e-12)
    assert np.allclose(d["m"], rho * math.pi * (g["diameter"] / 2) ** 2 * g["length"], rtol=1e-12)
    assert 0.55 < (g["length"] / spec.length).min() and (g["length"] / spec.length).max() < 1.45
    for a in range(spec.n_apples):                       # apples sit at the tip (0, 0, L): they stay at the new tip
        b = spec.apple_link[a]
        assert abs(g["apple_offset"][a][2] - g["length"][b]) < 1e-6 * g["length"][b]
    R, p, _, _ = w.fk()
    s = w.get_state()
    for a in range(spec.n_apples):
        b = spec.apple_link[a]
        xh = p[b] + R[b] @ g["apple_offset"][a]
        assert np.allclose(xh - s["apple_x"][a], [0, 0, float(spec.apple_mass[a]) * G / float(spec.apple_k[a])], atol=1e-9)


def test_geometry_randomization_lean_twist_spread_against_scipy():
    """Lean tilts the trunk by the drawn angle about a horizontal axis of drawn azimuth; twist turns every child about
    its parent's axis; spread scales the angle between a child and its parent's axis and keeps its azimuth."""
    spec = binary_tree_config1()
    seed = 4242
    key = [seed, 0]
    Q0 = np.stack([Rotation.from_quat([q[1], q[2], q[3], q[0]]).as_matrix() for q in spec.rest_quat.astype(np.float64)])
    w = OracleWorld(spec, config_params(1), world_index=2)
    o0, o1 = philox4x32_10([2, 0, 3, 0], key), philox4x32_10([2, 1, 3, 0], key)
    # lean only
    w.randomize_geometry(seed, lean=(0.05, 0.30))
    lean = float(_u32_uniform(o0[1], 0.05, 0.30)); phi = float(_u32_uniform(o1[0], 0.0, 6.2831855))
    Q = w.geometry()["Q"]
    Rl = Rotation.from_rotvec(lean * np.array([math.cos(phi), math.sin(phi), 0.0])).as_matrix()
    assert np.abs(Q[0] - Rl @ Q0[0]).max() < 1e-12 and np.abs(Q[1:] - Q0[1:]).max() < 1e-12
    assert abs(math.acos(np.clip((Q[0] @ [0, 0, 1]) @ (Q0[0] @ [0, 0, 1]), -1, 1)) - lean) < 1e-9
    # twist only
    w.randomize_geometry(seed, twist=(-0.6, 0.6))
    tw = float(_u32_uniform(o0[3], -0.6, 0.6))
    Q = w.geometry()["Q"]
    Rz = Rotation.from_euler("z", tw).as_matrix()
    assert abs(tw) > 1e-3 and np.abs(Q[0] - Q0[0]).max() < 1e-15
    for i in range(1, spec.n_links):
        assert np.abs(Q[i] - Rz @ Q0[i]).max() < 1e-12
    # spread only
    w.randomize_geometry(seed, spread=(0.1, 0.4))
    sp = float(_u32_uniform(o0[2], 0.1, 0.4))
    Q = w.geometry()["Q"]
    for i in range(1, spec.n_links):
        d0, d1 = Q0[i] @ [0, 0, 1], Q[i] @ [0, 0, 1]
        a0, a1 = math.atan2(math.hypot(d0[0], d0[1]), d0[2]), math.atan2(math.hypot(d1[0], d1[1]), d1[2])
        assert abs(a1 - (1 + sp) * a0) < 1e-9 and abs(math.atan2(d1[1], d1[0]) - math.atan2(d0[1], d0[0])) < 1e-9
        assert abs(np.linalg.det(Q[i]) - 1) < 1e-12 and np.abs(Q[i] @ Q[i].T - np.eye(3)).max() < 1e-12


def test_geometry_randomization_droop_compounds_per_internode():
    """"a gravimorphic droop multiplier applied inside a forward-kinematic re-walk so droop compounds per
    internode".  A straight chain inclined by theta_0: internode k ends up at theta_k = t + droop sin t with
    t = theta_(k-1) (its parent's final inclination), in the plane of the chain."""
    n, th0, droop = 6, math.radians(40.0), 0.15
    spec = chain_spec(n, 1.2, 0.03, root_quat=quat_axis("x", -math.degrees(th0)))     # tilted in the y-z plane
    w = OracleWorld(spec, Params(), world_index=0)
    R, p, _, _ = w.fk()
    th0 = math.acos(R[0][2, 2])                        # the inputs are fp32: the inclination and the multiplier as
    droop = float(np.float32(droop))                   # the oracle receives them
    w.randomize_geometry(1, droop=(droop, droop))
    R, p, _, _ = w.fk()
    t = 0.0
    prev = th0
    for k in range(n):
        base = prev if k > 0 else th0
        t = base + droop * math.sin(base)
        d = R[k] @ [0, 0, 1]
        assert abs(d[0]) < 1e-12 and d[1] > 0                          # stays in the plane it was tilted in
        assert abs(math.acos(np.clip(d[2], -1, 1)) - t) < 1e-9, (k, t)
        prev = t
    assert prev > th0 + n * droop * math.sin(th0) * 0.99              # compounding: more than n equal increments


# ---------------------------------------------------------------- post-rupture dissipation and the force rails (8(f) item 1)
def test_post_rupture_coulomb_friction_stops_a_free_hinge_in_the_closed_form_time():
    """A34: a ruptured joint carries a friction torque T_f = fric_frac M_max against its velocity, taken
    as the damper T_f / |qd| at the start-of-step speed.  One free hinge, no gravity: (J + h T / |w|) w+ = J w, i.e.
    w+ = w - h T / J to first order: it stops after J w0 / T.  With the ramp T grows linearly to fric_ramp T_0 over
    fric_time, counted from the step of the rupture."""
    L, d, rho, MOR = 0.5, 0.02, 800.0, 60e6
    spec = chain_spec(1, L, d)
    Lf, df = float(spec.length[0]), float(spec.diameter[0])
    m = rho * math.pi * (df / 2) ** 2 * Lf
    J = m * Lf * Lf / 3 + m * (df / 2) ** 2 / 4
    Mmax = MOR * math.pi * df ** 3 / 32
    h = float(np.float32(1e-3))
    for ramp, t_r in ((1.0, 1.5), (5.0, 0.05)):
        frac = float(np.float32(2e-4))
        P = Params(h=1e-3, gravity=(0, 0, 0), qd_max=0.0, fric_frac=frac, fric_ramp=ramp, fric_time=t_r, fric_veps=1e-3)
        w = OracleWorld(spec, P)
        w0 = 3.0
        w.set_state(qd=[w0, 0.0], ruptured=[1])
        v, steps, hist = w0, 0, []
        T0 = frac * Mmax
        t_rf = float(np.float32(t_r))
        while v > 2e-3 and steps < 4000:
            T = T0 * (1.0 + (ramp - 1.0) * min(h * steps / t_rf, 1.0))
            v = J * v / (J + h * T / max(v, float(np.float32(1e-3))))
            w.step(1)
            steps += 1
            assert abs(w.get_state()["qd"][0] - v) < 1e-9 * w0, (ramp, steps)
            hist.append(v)
        assert abs(w.get_state()["qd"][1]) < 1e-14
        if ramp == 1.0:                                    # constant torque: linear deceleration, stop at J w0 / T
            assert abs(steps * h - J * w0 / T0) < 0.02 * J * w0 / T0 + 3 * h, (steps * h, J * w0 / T0)
        else:                                              # the ramp shortens it
            assert steps * h < 0.75 * J * w0 / T0
    # an intact joint feels none of it
    wa, wb = OracleWorld(chain_spec(3, 0.9, 0.02), Params(fric_frac=0.1)), OracleWorld(chain_spec(3, 0.9, 0.02), Params())
    for x in (wa, wb):
        x.set_state(q=[0.01, 0.02, -0.01, 0.0, 0.02, 0.01], qd=[0.3, -0.2, 0.1, 0.5, -0.4, 0.2])
    assert np.array_equal(wa.system()[0], wb.system()[0]) and np.array_equal(wa.system()[1], wb.system()[1])


def test_snapped_subtree_drag_is_reduced():
    """A35 ("a snapped sub-tree's linear drag is also reduced"): alpha_i = mass_damping snap_drag_scale on
    the links at or below a ruptured joint.  A free hinge decays as v0 / (1 + h alpha scale)^n; the intact part of the
    tree keeps the full alpha: the system of a 2-link chain with the outer joint ruptured equals
    M + h alpha (M - M_outer) + h alpha scale M_outer, with M_outer the mass matrix of the outer link alone."""
    alpha, scale, h = 2.0, 0.2, float(np.float32(2e-3))
    spec = chain_spec(1, 0.5, 0.02)
    w = OracleWorld(spec, Params(gravity=(0, 0, 0), qd_max=0.0, mass_damping=alpha, snap_drag_scale=scale))
    w.set_state(qd=[0.7, 0.0], ruptured=[1])             # about the first axis only: theta_2 stays 0, M_11 constant
    sc = float(np.float32(scale))
    for n in range(1, 30):
        w.step(1)
        assert np.abs(w.get_state()["qd"] - np.array([0.7, 0.0]) / (1 + h * alpha * sc) ** n).max() < 1e-12
    spec2 = chain_spec(2, 0.8, 0.02)
    q = [0.05, -0.02, 0.03, 0.04]
    full = OracleWorld(spec2, Params(gravity=(0, 0, 0)))
    full.set_state(q=q, ruptured=[0, 1])
    M = full.mass_matrix()
    A0 = full.system()[0]
    # M_outer: the same chain with the inner link's inertia removed = M - M(inner only); M(inner only) touches DoF 0, 1
    inner = OracleWorld(chain_spec(1, 0.4, 0.02), Params(gravity=(0, 0, 0)))
    inner.set_state(q=q[:2])
    M_inner = np.zeros((4, 4)); M_inner[:2, :2] = inner.mass_matrix()
    M_outer = M - M_inner
    damped = OracleWorld(spec2, Params(gravity=(0, 0, 0), mass_damping=alpha, snap_drag_scale=scale))
    damped.set_state(q=q, ruptured=[0, 1])
    A1 = damped.system()[0]
    expect = A0 + h * alpha * M_inner + h * alpha * sc * M_outer
    assert np.abs(A1 - expect).max() < 1e-12 * np.abs(A1).max()


def test_force_rails_on_a_free_apple_and_never_on_static_loading():
    """A36 (App. B): (1) impulse cap: an applied force may not take a free body past rail_speed in one
    step; (2) power fade: the part of the force along the body's velocity fades out between rail_fade rail_speed and
    rail_speed; (3) speed brake above rail_speed.  A detached apple is the free body; gravity off."""
    mA, vl, brake = 0.2, 4.0, 50.0
    spec = chain_spec(1, 0.5, 0.02, apples=[(0, (0, 0, 0.5), mA, 2e3, 20.0)])
    h = float(np.float32(1e-3))
    mAf = float(np.float32(mA))
    P = Params(h=1e-3, gravity=(0, 0, 0), rail_speed=vl, rail_fade=0.5, rail_brake=brake)

    def run(v0, F, P=P):
        w = OracleWorld(spec, P)
        w.set_state(attached=[0], apple_v=[v0])
        w.apply_wrench(1, (0, 0, 0), F)
        w.step(1)
        return w.get_state()["apple_v"][0]
    # (1) cap: 5000 N on 0.2 kg would give 25 m/s in a step; the rail stops it at the limit, along the force
    assert np.allclose(run([0, 0, 0], (5000.0, 0, 0)), [vl, 0, 0], atol=1e-12)
    assert np.allclose(run([1.0, 0, 0], (0, 5000.0, 0)), [1.0, vl, 0], atol=1e-12)          # v . F^ = 0: full headroom
    # no effect below the cap and below the fade onset
    assert np.allclose(run([1.0, 0, 0], (30.0, 10.0, 0)), [1.0 + h * 30 / mAf, h * 10 / mAf, 0], atol=1e-12)
    # (2) fade: at 3 m/s (half way between onset 2 and limit 4) the parallel part is halved, the rest untouched
    assert np.allclose(run([3.0, 0, 0], (30.0, 10.0, 0)), [3.0 + h * 15 / mAf, h * 10 / mAf, 0], atol=1e-12)
    assert np.allclose(run([3.0, 0, 0], (-30.0, 10.0, 0)), [3.0 - h * 30 / mAf, h * 10 / mAf, 0], atol=1e-12)   # braking force: no fade
    # (3) brake above the limit: the pushing part is gone, and - brake m (|v| - v_lim) v^ acts
    assert np.allclose(run([6.0, 0, 0], (30.0, 0.0, 0)), [6.0 - h * brake * 2.0, 0, 0], atol=1e-12)
    # rails off: the raw force
    assert np.allclose(run([0, 0, 0], (5000.0, 0, 0), dataclasses.replace(P, rail_speed=0.0)), [h * 5000 / mAf, 0, 0], atol=1e-9)
    # the detach predicate sees the pull itself, not the railed force: config 1 with rails on has the same events, and
    # static loading of the connected tree is untouched (same state after the run)
    spec1 = binary_tree_config1()
    res = []
    for rs in (0.0, 3.0):
        w = OracleWorld(spec1, dataclasses.replace(config_params(1), rail_speed=rs))
        for s in range(400):
            for (_, body, pt, f) in config1_loads(spec1, s, 500, 30.0, 400.0):
                w.apply_wrench(body, pt, f)
            w.step(1)
        res.append((w.events(), w.get_state()["q"]))
    assert [e[:4] for e in res[0][0]] == [e[:4] for e in res[1][0]] and len(res[0][0]) == 1
    assert np.abs(res[0][1] - res[1][1]).max() < 1e-6
    # a rail so tight that it caps a 25 N pull to 1 N: path A still counts the pull itself (25 N > 20 N for 3 steps)
    w = OracleWorld(spec1, dataclasses.replace(config_params(1), rail_speed=0.01))
    w.apply_wrench(spec1.n_links + 2, (0, 0, 0), (0.0, 25.0, 0.0))
    w.step(4)
    ev = w.events()
    assert len(ev) == 1 and ev[0][1:4] == (2, 1, 2) and ev[0][4] == 25.0


# ---------------------------------------------------------------- round 3: the hysteresis resets, snapped sub-trees, the order of the
# updates inside a step, the absolute-velocity damper (the seven one-line mutants of round 2's review that survived)
def _pinned_link(nr, **kw):
    """One link whose joint an armature of 1e9 kg m^2 holds in place: q is whatever set_state puts there."""
    spec = chain_spec(1, 0.5, 0.02, armature=np.full((1, 2), 1e9, dtype=np.float32))
    d, L = float(spec.diameter[0]), float(spec.length[0])
    Mmax, K = 60e6 * math.pi * d ** 3 / 32, 8e9 * math.pi * d ** 4 / (64 * L)
    return spec, OracleWorld(spec, Params(gravity=(0, 0, 0), rupture_frames=nr, **kw)), Mmax / K


def test_rupture_counter_resets_on_a_miss():
    """PAPER.md:139 "N-frame hysteresis", reading A7: the N_r steps above M_max must be CONSECUTIVE.  Above for
    N_r - 1 steps, one step below, above again: the joint ruptures N_r steps after the SECOND crossing.
    (Perturbation this fails on: the counter kept, or merely not incremented, on a miss -- fires at step 3.)"""
    nr = 3
    spec, w, th = _pinned_link(nr)
    hi, lo = [0.6 * 1.01 * th, 0.8 * 1.01 * th], [0.6 * 0.99 * th, 0.8 * 0.99 * th]
    w.set_state(q=hi); w.step(nr - 1)                       # steps 0, 1: above
    assert w.get_counters()[0][0] == nr - 1
    w.set_state(q=lo); w.step(1)                            # step 2: below
    assert w.get_counters()[0][0] == 0 and w.events() == []
    w.set_state(q=hi); w.step(nr - 1)                       # steps 3, 4: above, not yet N_r in a row
    assert w.events() == [] and w.get_state()["ruptured"][0] == 0
    w.step(1)                                               # step 5
    ev = w.events()
    assert len(ev) == 1 and ev[0][1:4] == (nr - 1 + 1 + nr - 1, 0, 0)
    assert w.get_state()["ruptured"][0] == 1


def _apple_on_a_pinned_link(**kw):
    mA, ks, fdet = 0.2, 2e3, 20.0
    spec = chain_spec(1, 0.5, 0.08, apples=[(0, (0, 0, 0.5), mA, ks, fdet)], armature=np.full((1, 2), 1e9, dtype=np.float32))
    return spec, OracleWorld(spec, Params(**kw)), mA, ks, fdet, np.array([0.0, 0.0, 0.5])


def test_pull_counter_resets_on_a_miss():
    """PAPER.md:163 "sustained for a few frames", reading A14, path A: pull above f_detach for 2 steps, 1 step below,
    then above: the apple detaches N_A = 3 steps after the SECOND onset, with value |f_user| and threshold f_detach.
    (Perturbation this fails on: c_A not reset on a miss -- detaches at step 3.)"""
    spec, w, mA, ks, fdet, _ = _apple_on_a_pinned_link(detach_frames_pull=3, detach_frames_tension=10 ** 6)
    pattern = [1.5, 1.5, 0.5, 1.5, 1.5, 1.5, 1.5]
    fired = []
    for s, f in enumerate(pattern):
        w.apply_wrench(1, (0, 0, 0), (0.6 * f * fdet, 0.0, -0.8 * f * fdet))
        w.step(1)
        fired += w.events()
        if s == 2:
            assert w.get_counters()[1][0] == 0
    assert len(fired) == 1 and fired[0][1:4] == (5, 1, 0)
    assert abs(fired[0][4] - 1.5 * fdet) < 1e-5 and abs(fired[0][5] - fdet) < 1e-9


def test_tension_counter_resets_on_a_miss():
    """Reading A14, path B: |f_s| = k_s |x - x_hang| above kappa f_detach for 9 steps, 1 step below, then above:
    detach N_B = 10 steps after the second onset (step 19), value k_s |x - x_hang|, threshold kappa f_detach.  The
    stretch is imposed through set_state before every step (which leaves the counters alone).
    (Perturbation this fails on: c_B not reset on a miss -- detaches at step 10.)"""
    spec, w, mA, ks, fdet, xh = _apple_on_a_pinned_link(detach_frames_pull=10 ** 6, detach_frames_tension=10)
    kap = float(np.float32(1.1))
    s_hi, s_lo = 1.2 * kap * fdet / ks, 0.5 * kap * fdet / ks
    fired = []
    for s in range(24):
        st = s_lo if s == 9 else s_hi
        w.set_state(apple_x=[xh + st * np.array([0.0, 0.6, -0.8])], apple_v=[[0, 0, 0]])
        w.step(1)
        fired += [(s,) + e for e in w.events()]
        if fired:
            break
        if s == 9:
            assert w.get_counters()[2][0] == 0
    assert len(fired) == 1 and fired[0][0] == 19 and fired[0][2:5] == (19, 1, 0)
    assert abs(fired[0][5] - ks * s_hi) < 1e-7 and abs(fired[0][6] - kap * fdet) < 1e-9   # 1e-9 armature drift


def test_detach_path_A_takes_precedence_when_both_paths_complete_in_one_step():
    """Reading A14: one flag flip, one event; when the pull path and the tension path complete in the same step the
    event carries path A's pair (|f_user|, f_detach).  (Perturbation: path B tested first.)"""
    spec, w, mA, ks, fdet, xh = _apple_on_a_pinned_link(detach_frames_pull=3, detach_frames_tension=3)
    kap = float(np.float32(1.1))
    st = 1.3 * kap * fdet / ks
    w.apply_wrench(1, (0, 0, 0), (0.0, 0.0, -1.5 * fdet))
    for s in range(3):
        w.set_state(apple_x=[xh + st * np.array([0.0, 0.0, -1.0])], apple_v=[[0, 0, 0]])
        assert w.events() == []
        w.step(1)
    rc, cA, cB = w.get_counters()
    assert cA[0] >= 3 and cB[0] >= 3                       # both paths complete in step 2
    ev = w.events()
    assert len(ev) == 1 and ev[0][1:4] == (2, 1, 0)
    assert abs(ev[0][4] - 1.5 * fdet) < 1e-5 and abs(ev[0][5] - fdet) < 1e-9
    assert w.get_state()["attached"][0] == 0


def test_snapped_flag_covers_the_whole_subtree_below_a_ruptured_joint():
    """PAPER.md:398 "forces off on snapped sub-trees", reading A10: with joint 1 of a 3-link chain ruptured, a wrench
    on link 2 (BELOW the break, itself intact) leaves b untouched when forces_off_on_snapped = 1 and adds exactly
    h J^T F when it is 0; a wrench on link 0 (above the break) always acts.
    (Perturbation this fails on: snapped_i = ruptured_i without the parent's flag.)"""
    spec = chain_spec(3, 0.9, 0.03, root_quat=quat_axis("y", 70.0))
    rng = np.random.default_rng(3)
    q = rng.uniform(-0.1, 0.1, size=6)
    pt, F = (0.01, -0.02, 0.2), np.array([1.5, -2.0, 0.7])
    h = float(np.float32(2e-3))

    def rhs(flag, body):
        w = OracleWorld(spec, Params(forces_off_on_snapped=flag))
        w.set_state(q=q, ruptured=[0, 1, 0])
        b0 = w.system()[1]
        if body is not None:
            w.apply_wrench(body, pt, F)
        return w.system()[1] - b0

    assert np.abs(rhs(1, 2)).max() == 0.0
    ptf = np.asarray(pt, dtype=np.float32).astype(np.float64)
    for flag, body in ((0, 2), (1, 0), (0, 0)):
        J = _fd_jacobian(spec, q, body, ptf)
        db = rhs(flag, body)
        assert np.abs(db - h * J.T @ F).max() < 1e-7 * np.abs(db).max(), (flag, body)


def test_rupture_predicate_reads_the_end_of_step_angle():
    """SURVEY.md 8(c) steps 6 and 8, reading A8 (Eq. 5 on the configuration the step produced): a single DoF driven
    so that K |theta| crosses M_max between q and q + h qd+ with N_r = 1.  The event belongs to step 0 and its value is
    K |q + h qd+| with qd+ from the closed-form 1-DoF step map of the pin above.
    (Perturbation this fails on: the predicate on the start-of-step q -- event one step late, other value.)"""
    L, d, rho, E, MOR = 0.6, 0.02, 800.0, 8e9, 60e6
    spec = chain_spec(1, L, d, density=rho, E=E, MOR=MOR)
    w = OracleWorld(spec, Params(h=2e-3, gravity=(0, 0, 0), rupture_frames=1, qd_max=0.0))
    hh, cd = float(np.float32(2e-3)), float(np.float32(0.05))
    r, Lf = float(spec.diameter[0]) / 2, float(spec.length[0])
    m = rho * math.pi * r * r * Lf
    J = m * Lf * Lf / 3 + m * r * r / 4
    K = E * math.pi * (2 * r) ** 4 / (64 * Lf)
    Mmax = MOR * math.pi * (2 * r) ** 3 / 32
    q0, v0 = 0.999 * Mmax / K, 20.0
    v1 = (J * v0 - hh * K * q0) / (J + hh * cd * K + hh * hh * K)
    q1 = q0 + hh * v1
    assert K * q0 < Mmax < K * q1                           # the crossing happens inside step 0
    w.set_state(q=[0.0, q0], qd=[0.0, v0])
    w.step(1)
    ev = w.events()
    assert len(ev) == 1 and ev[0][1:4] == (0, 0, 0)
    assert abs(ev[0][4] - K * q1) < 1e-9 * K * q1 and abs(ev[0][5] - Mmax) < 1e-9 * Mmax
    assert abs(w.get_state()["q"][1] - q1) < 1e-13


def test_apple_position_advances_with_the_end_of_step_velocity():
    """PAPER.md:151 (3-DoF fruit): semi-implicit Euler, v += h a, then x += h v with the NEW v.
    A detached apple under gravity and a constant pull: x_n = x_0 + h^2 a n (n + 1) / 2 exactly.
    (Perturbation this fails on: x += h v_old, which gives n (n - 1) / 2 and misses by h^2 a n.)"""
    mA = 0.25
    spec = chain_spec(1, 0.5, 0.08, apples=[(0, (0, 0, 0.5), mA, 2e3, 20.0)])
    w = OracleWorld(spec, Params(h=2e-3))
    hh = float(np.float32(2e-3))
    w.set_state(attached=[0])
    x0 = w.get_state()["apple_x"][0].copy()
    F = np.asarray(np.float32([0.3, -0.2, 0.9]), dtype=np.float64)
    w.apply_wrench(1, (0, 0, 0), F)
    a = np.array([0.0, 0.0, -G]) + F / float(np.float32(mA))
    n = 25
    w.step(n)
    s = w.get_state()
    assert np.abs(s["apple_v"][0] - hh * a * n).max() < 1e-12
    assert np.abs(s["apple_x"][0] - (x0 + hh * hh * a * n * (n + 1) / 2)).max() < 1e-12
    assert np.linalg.norm(hh * hh * a * n) > 1e-4           # the size of the miss of the start-of-step variant


def test_tether_damper_acts_on_the_absolute_apple_velocity():
    """Eq. 6, reading A11: f = -k_s (x - x_hang) - c_s v with v the apple's own (world) velocity.
    (a) the branch swings (armature keeps qd), the apple is at rest in the world: after one step its velocity is
    h (g - k_s (x - x_hang) / m), no damper term although the hang point moves at |v_hang| = 0.5 m/s;
    (b) the branch is at rest, the apple moves: the damper term is -c_s v / m.
    (Perturbation this fails on: the damper on the velocity relative to the hang point.)"""
    mA, ks, zeta = 0.2, 2e3, 0.1
    spec = chain_spec(1, 0.5, 0.08, apples=[(0, (0, 0, 0.5), mA, ks, 1e6)], armature=np.full((1, 2), 1e9, dtype=np.float32))
    hh = float(np.float32(2e-3))
    m32, k32 = float(np.float32(mA)), float(np.float32(ks))
    cs = OracleWorld(spec, Params(zeta_s=zeta)).material()["c"][0]
    assert abs(cs - 2 * float(np.float32(zeta)) * math.sqrt(k32 * m32)) < 1e-9
    xh = np.array([0.0, 0.0, 0.5])
    dx = np.array([0.004, -0.003, -0.006])
    g = np.array([0.0, 0.0, -G])
    for qd, v in (([1.0, 0.0], np.zeros(3)), ([0.0, 0.0], np.array([0.3, -0.2, 0.1]))):
        w = OracleWorld(spec, Params(zeta_s=zeta))
        w.set_state(qd=qd, apple_x=[xh + dx], apple_v=[v])
        w.step(1)
        v1 = w.get_state()["apple_v"][0]
        assert np.abs(v1 - (v + hh * (g - k32 * dx / m32 - cs * v / m32))).max() < 1e-12, (qd, v1)
    assert hh * cs * 0.5 / m32 > 1e-3                        # what the relative-velocity variant would add in (a)
