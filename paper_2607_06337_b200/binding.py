"""Thin ctypes binding of the C ABI in include/orchard.h (same names, argument
marshalling only).  PyTorch supplies device memory (the workspace) and the CUDA
stream; nothing is computed here.  There is no CPU fallback: if libob.so is
missing or no CUDA device is present, construction fails loudly."""
from __future__ import annotations

import ctypes as C
import os
from typing import List, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libob.so")

OB_OK, OB_E_ARG, OB_E_CAPACITY, OB_E_WORKSPACE, OB_E_CUDA = 0, -1, -2, -3, -4
OB_MAX_WRENCH = 8
OB_STATUS_NONFINITE, OB_STATUS_CG_MAXITER = 1, 2

EXPORTS = [
    "ob_default_params", "ob_workspace_bytes", "ob_create", "ob_randomize", "ob_apply_wrench",
    "ob_apply_wrench_batch", "ob_step", "ob_get_state", "ob_set_state", "ob_get_apple_x64", "ob_get_counters", "ob_set_counters",
    "ob_get_material", "ob_events", "ob_stats", "ob_launch_info", "ob_last_error", "ob_destroy",
    "ob_sizeof_params", "ob_sizeof_world_spec", "ob_sizeof_event", "ob_counters", "ob_flush",
    "ob_selftest_philox", "ob_get_state_batch", "ob_set_apple_x64", "ob_set_step", "ob_get_counters_batch",
    "ob_get_material_batch", "ob_world_blob_bytes", "ob_save_world", "ob_load_world", "ob_iter_histogram",
    "ob_randomize_geometry", "ob_get_geometry", "ob_sizeof_geometry_ranges", "ob_get_rupture_steps",
    "ob_set_rupture_steps", "ob_selftest_philox_static",
]


class ob_world_spec(C.Structure):
    _fields_ = [
        ("n_links", C.c_int32), ("parent", C.c_void_p), ("length", C.c_void_p), ("diameter", C.c_void_p),
        ("rest_quat", C.c_void_p), ("armature", C.c_void_p),
        ("density", C.c_float), ("E", C.c_float), ("MOR", C.c_float),
        ("n_apples", C.c_int32), ("apple_link", C.c_void_p), ("apple_offset", C.c_void_p),
        ("apple_mass", C.c_void_p), ("apple_radius", C.c_void_p), ("apple_k", C.c_void_p),
        ("apple_c", C.c_void_p), ("apple_detach", C.c_void_p),
    ]


class ob_params(C.Structure):
    _fields_ = [
        ("h", C.c_float), ("gravity", C.c_float * 3), ("c_d", C.c_float), ("cg_tol", C.c_float),
        ("cg_max_iter", C.c_int32), ("precond", C.c_int32), ("cg_norm", C.c_int32), ("rupture_frames", C.c_int32),
        ("detach_frames_pull", C.c_int32), ("detach_kappa", C.c_float), ("detach_frames_tension", C.c_int32),
        ("react_max", C.c_float), ("tether_implicit", C.c_int32), ("qd_max", C.c_float), ("zeta_s", C.c_float),
        ("forces_off_on_snapped", C.c_int32),
        ("range_E", C.c_float * 2), ("range_MOR", C.c_float * 2), ("range_density", C.c_float * 2),
        ("range_detach", C.c_float * 2), ("range_apple_mass", C.c_float * 2), ("mass_damping", C.c_float),
        ("fric_frac", C.c_float), ("fric_ramp", C.c_float), ("fric_time", C.c_float), ("fric_veps", C.c_float),
        ("snap_drag_scale", C.c_float), ("rail_speed", C.c_float), ("rail_fade", C.c_float), ("rail_brake", C.c_float),
    ]


class ob_geometry_ranges(C.Structure):
    _fields_ = [(n, C.c_float * 2) for n in ("droop", "lean", "spread", "twist", "scale_length", "scale_diameter",
                                             "jitter_length", "jitter_diameter")]


GEOMETRY_IDENTITY = dict(droop=(0.0, 0.0), lean=(0.0, 0.0), spread=(0.0, 0.0), twist=(0.0, 0.0),
                         scale_length=(1.0, 1.0), scale_diameter=(1.0, 1.0), jitter_length=(1.0, 1.0),
                         jitter_diameter=(1.0, 1.0))


class ob_event(C.Structure):
    _fields_ = [("world", C.c_int32), ("step", C.c_int32), ("kind", C.c_int32), ("index", C.c_int32),
                ("value", C.c_float), ("threshold", C.c_float)]


_lib = None


def load_library():
    """dlopen libob.so (built in-tree by paper_2607_06337_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2607_06337_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i32, u64 = C.c_void_p, C.c_int, C.c_uint64
        L.ob_default_params.argtypes = [C.POINTER(ob_params)]
        L.ob_workspace_bytes.argtypes = [vp, i32, C.POINTER(ob_params), C.POINTER(C.c_size_t)]
        L.ob_create.argtypes = [vp, i32, C.POINTER(ob_params), vp, C.c_size_t, vp, C.POINTER(vp)]
        L.ob_randomize.argtypes = [vp, u64]
        L.ob_apply_wrench.argtypes = [vp, i32, i32, vp, vp]
        L.ob_apply_wrench_batch.argtypes = [vp, i32, vp, vp, vp, vp]
        L.ob_step.argtypes = [vp, i32]
        L.ob_flush.argtypes = [vp]
        L.ob_get_state.argtypes = [vp, i32] + [vp] * 8
        L.ob_set_state.argtypes = [vp, i32] + [vp] * 6
        L.ob_get_apple_x64.argtypes = [vp, i32, vp]
        L.ob_set_apple_x64.argtypes = [vp, i32, vp]
        L.ob_set_step.argtypes = [vp, i32, C.c_int32]
        L.ob_get_rupture_steps.argtypes = [vp, i32, vp]
        L.ob_set_rupture_steps.argtypes = [vp, i32, vp]
        L.ob_get_state_batch.argtypes = [vp, i32, i32] + [vp] * 8
        L.ob_get_counters_batch.argtypes = [vp, i32, i32] + [vp] * 3
        L.ob_get_material_batch.argtypes = [vp, i32, i32] + [vp] * 3
        L.ob_world_blob_bytes.argtypes = [vp, i32, C.POINTER(C.c_size_t)]
        L.ob_save_world.argtypes = [vp, i32, vp, C.c_size_t]
        L.ob_load_world.argtypes = [vp, i32, vp, C.c_size_t]
        L.ob_iter_histogram.argtypes = [vp, vp, i32, i32]
        L.ob_randomize_geometry.argtypes = [vp, u64, C.POINTER(ob_geometry_ranges)]
        L.ob_get_geometry.argtypes = [vp, i32] + [vp] * 4
        L.ob_get_counters.argtypes = [vp, i32] + [vp] * 3
        L.ob_set_counters.argtypes = [vp, i32] + [vp] * 3
        L.ob_get_material.argtypes = [vp, i32] + [vp] * 3
        L.ob_events.argtypes = [vp, vp, i32, C.POINTER(C.c_int)]
        L.ob_stats.argtypes = [vp, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64), C.POINTER(C.c_int32)]
        L.ob_launch_info.argtypes = [vp] + [C.POINTER(C.c_int32)] * 4
        L.ob_counters.argtypes = [vp, C.POINTER(C.c_uint64 * 4)]
        L.ob_selftest_philox.argtypes = [i32] + [vp] * 6
        L.ob_selftest_philox_static.argtypes = [i32] + [vp] * 5
        L.ob_last_error.argtypes = [vp]
        L.ob_last_error.restype = C.c_char_p
        L.ob_destroy.argtypes = [vp]
        L.ob_destroy.restype = None
        for name in ("ob_sizeof_params", "ob_sizeof_world_spec", "ob_sizeof_event", "ob_sizeof_geometry_ranges"):
            getattr(L, name).argtypes = []
        for name in EXPORTS:
            if name not in ("ob_last_error", "ob_destroy"):
                getattr(L, name).restype = C.c_int
        if (L.ob_sizeof_params(), L.ob_sizeof_world_spec(), L.ob_sizeof_event()) != (
                C.sizeof(ob_params), C.sizeof(ob_world_spec), C.sizeof(ob_event)) or \
                L.ob_sizeof_geometry_ranges() != C.sizeof(ob_geometry_ranges):
            raise RuntimeError("libob.so was built from a different include/orchard.h than this binding")
        _lib = L
    return _lib


class OrchardError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"orchard error {code}: {msg}")
        self.code = code


def default_params() -> ob_params:
    p = ob_params()
    rc = load_library().ob_default_params(C.byref(p))
    if rc != OB_OK:
        raise OrchardError(rc, "ob_default_params")
    return p


def params_struct(p) -> ob_params:
    """workloads.Params (plain data) -> ob_params."""
    s = default_params()
    s.h = p.h
    s.gravity = (C.c_float * 3)(*p.gravity)
    for name in ("c_d", "cg_tol", "cg_max_iter", "precond", "cg_norm", "rupture_frames", "detach_frames_pull", "detach_kappa",
                 "detach_frames_tension", "react_max", "tether_implicit", "qd_max", "zeta_s",
                 "forces_off_on_snapped", "mass_damping", "fric_frac", "fric_ramp", "fric_time", "fric_veps",
                 "snap_drag_scale", "rail_speed", "rail_fade", "rail_brake"):
        setattr(s, name, getattr(p, name))
    for name in ("range_E", "range_MOR", "range_density", "range_detach", "range_apple_mass"):
        setattr(s, name, (C.c_float * 2)(*getattr(p, name)))
    return s


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _ptr(a):
    return None if a is None else a.ctypes.data


def marshal_specs(specs: Sequence) -> tuple:
    """workloads.WorldSpec list -> (ob_world_spec array, keep-alive list)."""
    arr = (ob_world_spec * len(specs))()
    keep = []
    for k, sp in enumerate(specs):
        par, ln, dm, qt = _i32(sp.parent), _f32(sp.length), _f32(sp.diameter), _f32(sp.rest_quat)
        arm = None if sp.armature is None else _f32(sp.armature)
        al, ao, am = _i32(sp.apple_link), _f32(sp.apple_offset), _f32(sp.apple_mass)
        ar, ak, ad = _f32(sp.apple_radius), _f32(sp.apple_k), _f32(sp.apple_detach)
        ac = None if sp.apple_c is None else _f32(sp.apple_c)
        keep += [par, ln, dm, qt, arm, al, ao, am, ar, ak, ad, ac]
        s = arr[k]
        s.n_links = int(par.shape[0])
        s.parent, s.length, s.diameter, s.rest_quat, s.armature = _ptr(par), _ptr(ln), _ptr(dm), _ptr(qt), _ptr(arm)
        s.density, s.E, s.MOR = float(sp.density), float(sp.E), float(sp.MOR)
        s.n_apples = int(al.shape[0])
        s.apple_link, s.apple_offset, s.apple_mass = _ptr(al), _ptr(ao), _ptr(am)
        s.apple_radius, s.apple_k, s.apple_c, s.apple_detach = _ptr(ar), _ptr(ak), _ptr(ac), _ptr(ad)
    return arr, keep


class Orchard:
    """One ob_ctx.  Methods carry the C names without the ob_ prefix."""

    def __init__(self, specs: Sequence, params, device: str = "cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: the orchard step has no CPU fallback")
        self._L = load_library()
        self.specs = list(specs)
        self.n_worlds = len(self.specs)
        self.n_links = [s.n_links for s in self.specs]
        self.n_apples = [s.n_apples for s in self.specs]
        self.params = params if isinstance(params, ob_params) else params_struct(params)
        arr, keep = marshal_specs(self.specs)
        nbytes = C.c_size_t(0)
        rc = self._L.ob_workspace_bytes(arr, self.n_worlds, C.byref(self.params), C.byref(nbytes))
        if rc != OB_OK:
            raise OrchardError(rc, self._L.ob_last_error(None).decode())
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.workspace = torch.empty(int(nbytes.value) + 256, dtype=torch.uint8, device=self.device)
        base = (self.workspace.data_ptr() + 255) // 256 * 256
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        h = C.c_void_p()
        rc = self._L.ob_create(arr, self.n_worlds, C.byref(self.params), C.c_void_p(base), nbytes,
                               C.c_void_p(self.stream.cuda_stream), C.byref(h))
        del keep
        if rc != OB_OK:
            raise OrchardError(rc, self._L.ob_last_error(None).decode())
        self._h = h

    # -- plumbing --
    def _check(self, rc: int):
        if rc != OB_OK:
            raise OrchardError(rc, self._L.ob_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None):
            self._L.ob_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the C calls --
    def randomize(self, seed: int):
        self._check(self._L.ob_randomize(self._h, C.c_uint64(seed)))

    def randomize_geometry(self, seed: int, **ranges):
        """ranges: any of GEOMETRY_IDENTITY's keys as (lo, hi); the others keep their identity value."""
        g = ob_geometry_ranges()
        for k, v in {**GEOMETRY_IDENTITY, **ranges}.items():
            setattr(g, k, (C.c_float * 2)(*v))
        self._check(self._L.ob_randomize_geometry(self._h, C.c_uint64(seed), C.byref(g)))

    def get_geometry(self, world: int) -> dict:
        N, A = self.n_links[world], self.n_apples[world]
        Ln = np.zeros(N, np.float32); dm = np.zeros(N, np.float32); q = np.zeros((N, 4), np.float64)
        ao = np.zeros((A, 3), np.float32)
        self._check(self._L.ob_get_geometry(self._h, world, _ptr(Ln), _ptr(dm), _ptr(q), _ptr(ao)))
        return dict(length=Ln, diameter=dm, rest_quat=q, apple_offset=ao)

    def apply_wrench(self, world: int, body: int, point, force):
        p, f = _f32(point), _f32(force)
        self._check(self._L.ob_apply_wrench(self._h, world, body, _ptr(p), _ptr(f)))

    def apply_wrench_batch(self, world, body, point3, force3):
        w, b, p, f = _i32(world), _i32(body), _f32(point3), _f32(force3)
        self._check(self._L.ob_apply_wrench_batch(self._h, int(w.shape[0]), _ptr(w), _ptr(b), _ptr(p), _ptr(f)))

    def flush(self):
        self._check(self._L.ob_flush(self._h))

    def step(self, n: int = 1):
        self._check(self._L.ob_step(self._h, n))

    def get_state(self, world: int, pose: bool = False) -> dict:
        if not pose:
            b = self.get_state_batch(world, 1)
            return dict(q=b["q"], qd=b["qd"], apple_x=b["apple_x"], apple_x64=b["apple_x64"], apple_v=b["apple_v"],
                        ruptured=b["ruptured"], attached=b["attached"], step=int(b["info"][0, 0]),
                        last_iters=int(b["info"][0, 1]), status=int(b["info"][0, 2]))
        N, A = self.n_links[world], self.n_apples[world]
        q = np.zeros(2 * N, np.float32); qd = np.zeros(2 * N, np.float32)
        ax = np.zeros((A, 3), np.float32); av = np.zeros((A, 3), np.float32)
        rup = np.zeros(N, np.uint8); att = np.zeros(A, np.uint8)
        pose7 = np.zeros((N, 7), np.float32)
        info = np.zeros(3, np.int32)
        self._check(self._L.ob_get_state(self._h, world, _ptr(q), _ptr(qd), _ptr(ax), _ptr(av), _ptr(rup), _ptr(att),
                                         _ptr(pose7), _ptr(info)))
        x64 = np.zeros((A, 3), np.float64)
        if A:
            self._check(self._L.ob_get_apple_x64(self._h, world, _ptr(x64)))
        return dict(q=q, qd=qd, apple_x=ax, apple_v=av, ruptured=rup, attached=att, link_pose7=pose7, apple_x64=x64,
                    step=int(info[0]), last_iters=int(info[1]), status=int(info[2]))

    def get_state_batch(self, world0: int = 0, n_worlds: Optional[int] = None, out: Optional[dict] = None) -> dict:
        """ob_get_state_batch: worlds [world0, world0 + n_worlds), outputs concatenated in world order.  `out` may be
        the dict of a previous call (same range): its arrays are reused."""
        n = self.n_worlds - world0 if n_worlds is None else n_worlds
        NL, NA = sum(self.n_links[world0:world0 + n]), sum(self.n_apples[world0:world0 + n])
        if out is None:
            out = dict(q=np.zeros(2 * NL, np.float32), qd=np.zeros(2 * NL, np.float32),
                       apple_x=np.zeros((NA, 3), np.float32), apple_x64=np.zeros((NA, 3), np.float64),
                       apple_v=np.zeros((NA, 3), np.float32), ruptured=np.zeros(NL, np.uint8),
                       attached=np.zeros(NA, np.uint8), info=np.zeros((n, 3), np.int32))
        self._check(self._L.ob_get_state_batch(self._h, world0, n, _ptr(out["q"]), _ptr(out["qd"]), _ptr(out["apple_x"]),
                                               _ptr(out["apple_x64"]), _ptr(out["apple_v"]), _ptr(out["ruptured"]),
                                               _ptr(out["attached"]), _ptr(out["info"])))
        return out

    def set_apple_x64(self, world: int, apple_x):
        x = np.ascontiguousarray(apple_x, dtype=np.float64)
        self._check(self._L.ob_set_apple_x64(self._h, world, _ptr(x)))

    def set_step(self, world: int, step: int):
        self._check(self._L.ob_set_step(self._h, world, int(step)))

    def get_rupture_steps(self, world: int) -> np.ndarray:
        r = np.zeros(self.n_links[world], np.int32)
        self._check(self._L.ob_get_rupture_steps(self._h, world, _ptr(r)))
        return r

    def set_rupture_steps(self, world: int, rupture_step):
        r = _i32(rupture_step)
        self._check(self._L.ob_set_rupture_steps(self._h, world, _ptr(r)))

    def save_world(self, world: int) -> bytes:
        n = C.c_size_t(0)
        self._check(self._L.ob_world_blob_bytes(self._h, world, C.byref(n)))
        buf = np.zeros(n.value, np.uint8)
        self._check(self._L.ob_save_world(self._h, world, _ptr(buf), n))
        return buf.tobytes()

    def load_world(self, world: int, blob: bytes):
        buf = np.frombuffer(blob, dtype=np.uint8).copy()
        self._check(self._L.ob_load_world(self._h, world, _ptr(buf), C.c_size_t(buf.size)))

    def get_counters_batch(self, world0: int = 0, n_worlds: Optional[int] = None):
        n = self.n_worlds - world0 if n_worlds is None else n_worlds
        NL, NA = sum(self.n_links[world0:world0 + n]), sum(self.n_apples[world0:world0 + n])
        rc = np.zeros(NL, np.int32); ca = np.zeros(NA, np.int32); cb = np.zeros(NA, np.int32)
        self._check(self._L.ob_get_counters_batch(self._h, world0, n, _ptr(rc), _ptr(ca), _ptr(cb)))
        return rc, ca, cb

    def get_material_batch(self, world0: int = 0, n_worlds: Optional[int] = None) -> dict:
        n = self.n_worlds - world0 if n_worlds is None else n_worlds
        NA = sum(self.n_apples[world0:world0 + n])
        emr = np.zeros((n, 3), np.float32); det = np.zeros(NA, np.float32); mass = np.zeros(NA, np.float32)
        self._check(self._L.ob_get_material_batch(self._h, world0, n, _ptr(emr), _ptr(det), _ptr(mass)))
        return dict(E=emr[:, 0], MOR=emr[:, 1], density=emr[:, 2], detach=det, mass=mass)

    def iter_histogram(self, n_bins: int = 64, reset: bool = False) -> np.ndarray:
        bins = np.zeros(n_bins, np.uint64)
        self._check(self._L.ob_iter_histogram(self._h, _ptr(bins), n_bins, 1 if reset else 0))
        return bins

    def set_state(self, world: int, q=None, qd=None, apple_x=None, apple_v=None, ruptured=None, attached=None):
        def f(a):
            return None if a is None else _f32(a)

        def b(a):
            return None if a is None else np.ascontiguousarray(a, dtype=np.uint8)
        arrs = [f(q), f(qd), f(apple_x), f(apple_v), b(ruptured), b(attached)]
        self._check(self._L.ob_set_state(self._h, world, *[_ptr(a) for a in arrs]))

    def get_counters(self, world: int):
        N, A = self.n_links[world], self.n_apples[world]
        rc = np.zeros(N, np.int32); ca = np.zeros(A, np.int32); cb = np.zeros(A, np.int32)
        self._check(self._L.ob_get_counters(self._h, world, _ptr(rc), _ptr(ca), _ptr(cb)))
        return rc, ca, cb

    def set_counters(self, world: int, rc, ca, cb):
        rc, ca, cb = _i32(rc), _i32(ca), _i32(cb)
        self._check(self._L.ob_set_counters(self._h, world, _ptr(rc), _ptr(ca), _ptr(cb)))

    def get_material(self, world: int) -> dict:
        A = self.n_apples[world]
        emr = np.zeros(3, np.float32); det = np.zeros(A, np.float32); mass = np.zeros(A, np.float32)
        self._check(self._L.ob_get_material(self._h, world, _ptr(emr), _ptr(det), _ptr(mass)))
        return dict(E=emr[0], MOR=emr[1], density=emr[2], detach=det, mass=mass)

    _EV_DTYPE = np.dtype([("world", np.int32), ("step", np.int32), ("kind", np.int32), ("index", np.int32),
                          ("value", np.float32), ("threshold", np.float32)])

    def events(self, cap: Optional[int] = None) -> List[tuple]:
        """Drain the device event list: (world, step, kind, index, value, threshold), sorted by the library."""
        cap = cap if cap is not None else sum(self.n_links) + sum(self.n_apples) + 64
        cap = max(cap, 1)
        buf = getattr(self, "_ev_buf", None)
        if buf is None or len(buf) < cap:                  # one reusable host buffer (argument marshalling only)
            buf = self._ev_buf = (ob_event * cap)()
        n = C.c_int(0)
        rc = self._L.ob_events(self._h, buf, cap, C.byref(n))
        out = np.frombuffer(buf, dtype=self._EV_DTYPE, count=n.value).tolist()
        self._check(rc)
        return out

    def stats(self) -> dict:
        it, ws, fl = C.c_uint64(0), C.c_uint64(0), C.c_int32(0)
        self._check(self._L.ob_stats(self._h, C.byref(it), C.byref(ws), C.byref(fl)))
        return dict(cg_iters_total=int(it.value), world_steps_total=int(ws.value), n_flagged=int(fl.value))

    def counters(self) -> dict:
        v = (C.c_uint64 * 4)()
        self._check(self._L.ob_counters(self._h, C.byref(v)))
        return dict(h2d_bytes=int(v[0]), d2h_bytes=int(v[1]), kernel_launches=int(v[2]), step_calls=int(v[3]))

    def launch_info(self) -> dict:
        v = [C.c_int32(0) for _ in range(4)]
        self._check(self._L.ob_launch_info(self._h, *[C.byref(x) for x in v]))
        return dict(n_launches=v[0].value, grid=v[1].value, block=v[2].value, smem_bytes=v[3].value)
