"""ctypes view of the fp64 CPU oracle (oracle/orchard_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs import this package.  It
shares nothing with paper_2607_06337_b200/ (the CUDA path) and does not import
it.  Argument marshalling only; every number is computed in the C file.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import List, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "orchard_oracle.c")
# ORCHARD_ORACLE_SANITIZE=1 (tests/test_sanitizers.py): the same source built with ASan + UBSan into a library of its
# own; the process must then run under LD_PRELOAD=libasan.so.
_SANITIZE = os.environ.get("ORCHARD_ORACLE_SANITIZE", "") == "1"
_LIB = os.path.join(_HERE, "liborchard_oracle_san.so" if _SANITIZE else "liborchard_oracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C, OpenMP over worlds)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        opt = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined",
               "-fno-omit-frame-pointer"] if _SANITIZE else ["-O2"]
        cmd = ["gcc"] + opt + ["-std=c11", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off",
                               "-o", _LIB, _SRC, "-lm"]
        subprocess.check_call(cmd)
    return _LIB


class OboParams(C.Structure):
    _fields_ = [
        ("h", C.c_double), ("g", C.c_double * 3), ("c_d", C.c_double), ("cg_tol", C.c_double),
        ("cg_max_iter", C.c_int32), ("solver", C.c_int32), ("rupture_frames", C.c_int32),
        ("detach_frames_pull", C.c_int32), ("detach_kappa", C.c_double),
        ("detach_frames_tension", C.c_int32), ("tether_implicit", C.c_int32),
        ("react_max", C.c_double), ("qd_max", C.c_double), ("zeta_s", C.c_double), ("alpha_m", C.c_double),
        ("forces_off_on_snapped", C.c_int32), ("pad_", C.c_int32),
        ("fric_frac", C.c_double), ("fric_ramp", C.c_double), ("fric_time", C.c_double), ("fric_veps", C.c_double),
        ("snap_drag_scale", C.c_double), ("rail_speed", C.c_double), ("rail_fade", C.c_double), ("rail_brake", C.c_double),
        ("range_E", C.c_float * 2), ("range_MOR", C.c_float * 2), ("range_density", C.c_float * 2),
        ("range_detach", C.c_float * 2), ("range_apple_mass", C.c_float * 2),
    ]


class OboGeometryRanges(C.Structure):
    _fields_ = [(n, C.c_float * 2) for n in ("droop", "lean", "spread", "twist", "scale_length", "scale_diameter",
                                             "jitter_length", "jitter_diameter")]


GEOMETRY_IDENTITY = dict(droop=(0.0, 0.0), lean=(0.0, 0.0), spread=(0.0, 0.0), twist=(0.0, 0.0),
                         scale_length=(1.0, 1.0), scale_diameter=(1.0, 1.0), jitter_length=(1.0, 1.0),
                         jitter_diameter=(1.0, 1.0))


class OboEvent(C.Structure):
    _fields_ = [("world", C.c_int32), ("step", C.c_int32), ("kind", C.c_int32), ("index", C.c_int32),
                ("value", C.c_double), ("threshold", C.c_double)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.obo_world_new.restype = C.c_void_p
        L.obo_world_new.argtypes = [C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                    C.c_float, C.c_float, C.c_float, C.c_int, C.c_void_p, C.c_void_p,
                                    C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(OboParams)]
        L.obo_world_free.argtypes = [C.c_void_p]
        L.obo_randomize.argtypes = [C.c_void_p, C.c_uint64]
        L.obo_randomize_geometry.argtypes = [C.c_void_p, C.c_uint64, C.POINTER(OboGeometryRanges)]
        L.obo_diag_geometry.argtypes = [C.c_void_p] + [C.c_void_p] * 4
        L.obo_apply_wrench.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
        L.obo_apply_wrench.restype = C.c_int
        L.obo_step.argtypes = [C.c_void_p, C.c_int]
        L.obo_step_many.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.obo_get_state.argtypes = [C.c_void_p] + [C.c_void_p] * 7
        L.obo_set_state.argtypes = [C.c_void_p] + [C.c_void_p] * 6
        L.obo_get_counters.argtypes = [C.c_void_p] + [C.c_void_p] * 3
        L.obo_set_counters.argtypes = [C.c_void_p] + [C.c_void_p] * 3
        L.obo_set_step.argtypes = [C.c_void_p, C.c_int]
        L.obo_get_rupture_steps.argtypes = [C.c_void_p, C.c_void_p]
        L.obo_set_rupture_steps.argtypes = [C.c_void_p, C.c_void_p]
        L.obo_set_solver.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_int]
        L.obo_events.argtypes = [C.c_void_p, C.c_void_p, C.c_int]
        L.obo_events.restype = C.c_int
        L.obo_n_events.argtypes = [C.c_void_p]
        L.obo_n_events.restype = C.c_int
        L.obo_diag_material.argtypes = [C.c_void_p] + [C.c_void_p] * 4
        L.obo_diag_derived.argtypes = [C.c_void_p] + [C.c_void_p] * 5
        L.obo_diag_fk.argtypes = [C.c_void_p] + [C.c_void_p] * 4
        L.obo_diag_mass.argtypes = [C.c_void_p, C.c_void_p]
        L.obo_diag_rnea.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]
        L.obo_diag_system.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.obo_diag_energy.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.obo_philox4x32_10.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.obo_sizeof_params.restype = C.c_int
        L.obo_sizeof_event.restype = C.c_int
        assert L.obo_sizeof_params() == C.sizeof(OboParams)
        assert L.obo_sizeof_event() == C.sizeof(OboEvent)
        _lib = L
    return _lib


def philox4x32_10(ctr: Sequence[int], key: Sequence[int]) -> np.ndarray:
    c = np.asarray(ctr, dtype=np.uint32)
    k = np.asarray(key, dtype=np.uint32)
    o = np.zeros(4, dtype=np.uint32)
    lib().obo_philox4x32_10(c.ctypes.data, k.ctypes.data, o.ctypes.data)
    return o


def _params_struct(p, solver: int = 0) -> OboParams:
    s = OboParams()
    s.h = p.h
    s.g = (C.c_double * 3)(*[float(np.float32(x)) for x in p.gravity])
    s.c_d = float(np.float32(p.c_d))
    s.cg_tol = p.cg_tol
    s.cg_max_iter = p.cg_max_iter
    s.solver = solver
    s.rupture_frames = p.rupture_frames
    s.detach_frames_pull = p.detach_frames_pull
    s.detach_kappa = float(np.float32(p.detach_kappa))
    s.detach_frames_tension = p.detach_frames_tension
    s.tether_implicit = p.tether_implicit
    s.react_max = float(np.float32(p.react_max))
    s.qd_max = float(np.float32(p.qd_max))
    s.zeta_s = float(np.float32(p.zeta_s))
    s.alpha_m = float(np.float32(getattr(p, "mass_damping", 0.0)))
    s.forces_off_on_snapped = p.forces_off_on_snapped
    for name in ("fric_frac", "fric_ramp", "fric_time", "fric_veps", "snap_drag_scale", "rail_speed", "rail_fade", "rail_brake"):
        setattr(s, name, float(np.float32(getattr(p, name))))
    s.h = float(np.float32(p.h))
    for name in ("range_E", "range_MOR", "range_density", "range_detach", "range_apple_mass"):
        setattr(s, name, (C.c_float * 2)(*getattr(p, name)))
    return s


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


class OracleWorld:
    """One world of the oracle.  `spec` is a workloads.WorldSpec, `params` a
    workloads.Params (plain data; fp32-representable values are used so that
    both implementations see the same numbers)."""

    def __init__(self, spec, params, world_index: int = 0, solver: int = 0):
        L = lib()
        self.spec = spec
        self.N = spec.n_links
        self.A = spec.n_apples
        self.n = 2 * self.N
        ps = _params_struct(params, solver)
        par = np.ascontiguousarray(spec.parent, dtype=np.int32)
        arm = None if spec.armature is None else _f32(spec.armature)
        ac = None if spec.apple_c is None else _f32(spec.apple_c)
        al = np.ascontiguousarray(spec.apple_link, dtype=np.int32)
        self._keep = [par, arm, ac, al]
        self.h = L.obo_world_new(
            world_index, self.N, par.ctypes.data, _f32(spec.length).ctypes.data, _f32(spec.diameter).ctypes.data,
            _f32(spec.rest_quat).ctypes.data, None if arm is None else arm.ctypes.data,
            float(spec.density), float(spec.E), float(spec.MOR), self.A, al.ctypes.data,
            _f32(spec.apple_offset).ctypes.data, _f32(spec.apple_mass).ctypes.data, _f32(spec.apple_k).ctypes.data,
            None if ac is None else ac.ctypes.data, _f32(spec.apple_detach).ctypes.data, C.byref(ps))
        if not self.h:
            raise ValueError("obo_world_new rejected the spec")

    def __del__(self):
        if getattr(self, "h", None):
            lib().obo_world_free(self.h)
            self.h = None

    def randomize(self, seed: int):
        lib().obo_randomize(self.h, C.c_uint64(seed))

    def randomize_geometry(self, seed: int, **ranges):
        """ranges: any of GEOMETRY_IDENTITY's keys as (lo, hi); the others keep their identity value."""
        g = OboGeometryRanges()
        for k, v in {**GEOMETRY_IDENTITY, **ranges}.items():
            setattr(g, k, (C.c_float * 2)(*v))
        lib().obo_randomize_geometry(self.h, C.c_uint64(seed), C.byref(g))

    def geometry(self):
        L = np.zeros(self.N); d = np.zeros(self.N); Q = np.zeros((self.N, 3, 3)); ao = np.zeros((self.A, 3))
        lib().obo_diag_geometry(self.h, L.ctypes.data, d.ctypes.data, Q.ctypes.data, ao.ctypes.data)
        return dict(length=L, diameter=d, Q=Q, apple_offset=ao)

    def apply_wrench(self, body: int, point, force):
        p = np.asarray(point, dtype=np.float32).astype(np.float64)
        f = np.asarray(force, dtype=np.float32).astype(np.float64)
        rc = lib().obo_apply_wrench(self.h, body, p.ctypes.data, f.ctypes.data)
        if rc != 0:
            raise RuntimeError(f"obo_apply_wrench rc={rc}")

    def step(self, n: int = 1):
        lib().obo_step(self.h, n)

    def get_state(self):
        q = np.zeros(self.n); qd = np.zeros(self.n)
        ax = np.zeros((self.A, 3)); av = np.zeros((self.A, 3))
        rup = np.zeros(self.N, dtype=np.uint8); att = np.zeros(self.A, dtype=np.uint8)
        info = np.zeros(3, dtype=np.int32)
        lib().obo_get_state(self.h, q.ctypes.data, qd.ctypes.data, ax.ctypes.data, av.ctypes.data,
                            rup.ctypes.data, att.ctypes.data, info.ctypes.data)
        return dict(q=q, qd=qd, apple_x=ax, apple_v=av, ruptured=rup, attached=att,
                    step=int(info[0]), last_iters=int(info[1]), status=int(info[2]))

    def set_state(self, q=None, qd=None, apple_x=None, apple_v=None, ruptured=None, attached=None):
        def d(a):
            return None if a is None else np.ascontiguousarray(a, dtype=np.float64)

        def b(a):
            return None if a is None else np.ascontiguousarray(a, dtype=np.uint8)
        arrs = [d(q), d(qd), d(apple_x), d(apple_v), b(ruptured), b(attached)]
        lib().obo_set_state(self.h, *[None if a is None else a.ctypes.data for a in arrs])

    def get_counters(self):
        rc = np.zeros(self.N, dtype=np.int32); ca = np.zeros(self.A, dtype=np.int32); cb = np.zeros(self.A, dtype=np.int32)
        lib().obo_get_counters(self.h, rc.ctypes.data, ca.ctypes.data, cb.ctypes.data)
        return rc, ca, cb

    def set_counters(self, rc, ca, cb):
        rc = np.ascontiguousarray(rc, dtype=np.int32); ca = np.ascontiguousarray(ca, dtype=np.int32)
        cb = np.ascontiguousarray(cb, dtype=np.int32)
        lib().obo_set_counters(self.h, rc.ctypes.data, ca.ctypes.data, cb.ctypes.data)

    def set_step(self, step: int):
        lib().obo_set_step(self.h, step)

    def get_rupture_steps(self):
        r = np.zeros(self.N, dtype=np.int32)
        lib().obo_get_rupture_steps(self.h, r.ctypes.data)
        return r

    def set_rupture_steps(self, rstep):
        r = np.ascontiguousarray(rstep, dtype=np.int32)
        lib().obo_set_rupture_steps(self.h, r.ctypes.data)

    def set_solver(self, solver: int, tol: float = 1e-12, max_iter: int = 10000):
        lib().obo_set_solver(self.h, solver, tol, max_iter)

    def events(self) -> List[tuple]:
        n = lib().obo_n_events(self.h)
        buf = (OboEvent * max(n, 1))()
        n = lib().obo_events(self.h, buf, n)
        return [(e.world, e.step, e.kind, e.index, e.value, e.threshold) for e in buf[:n]]

    # ---- diagnostics used by the pins ----
    def material(self):
        emr = np.zeros(3, dtype=np.float32)
        adet = np.zeros(self.A); am = np.zeros(self.A); ac = np.zeros(self.A)
        lib().obo_diag_material(self.h, emr.ctypes.data, adet.ctypes.data, am.ctypes.data, ac.ctypes.data)
        return dict(E=emr[0], MOR=emr[1], density=emr[2], detach=adet, mass=am, c=ac)

    def derived(self):
        out = [np.zeros(self.N) for _ in range(5)]
        lib().obo_diag_derived(self.h, *[o.ctypes.data for o in out])
        return dict(K=out[0], Mmax=out[1], m=out[2], Ixx=out[3], Izz=out[4])

    def fk(self):
        R = np.zeros((self.N, 3, 3)); p = np.zeros((self.N, 3)); a1 = np.zeros((self.N, 3)); a2 = np.zeros((self.N, 3))
        lib().obo_diag_fk(self.h, R.ctypes.data, p.ctypes.data, a1.ctypes.data, a2.ctypes.data)
        return R, p, a1, a2

    def mass_matrix(self):
        M = np.zeros((self.n, self.n))
        lib().obo_diag_mass(self.h, M.ctypes.data)
        return M

    def rnea(self, qdd=None, use_gravity=True):
        qdd = np.zeros(self.n) if qdd is None else np.ascontiguousarray(qdd, dtype=np.float64)
        tau = np.zeros(self.n)
        lib().obo_diag_rnea(self.h, qdd.ctypes.data, 1 if use_gravity else 0, tau.ctypes.data)
        return tau

    def system(self):
        A = np.zeros((self.n, self.n)); b = np.zeros(self.n)
        lib().obo_diag_system(self.h, A.ctypes.data, b.ctypes.data)
        return A, b

    def energy(self):
        T = C.c_double(); V = C.c_double()
        lib().obo_diag_energy(self.h, C.byref(T), C.byref(V))
        return T.value, V.value


def step_many(worlds: Sequence[OracleWorld], n: int = 1):
    arr = (C.c_void_p * len(worlds))(*[w.h for w in worlds])
    lib().obo_step_many(arr, len(worlds), n)
