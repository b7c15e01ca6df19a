"""CPU-side checks of the C ABI (include/orchard.h): the library loads, exports every declared symbol,
its structs have the layout the binding assumes, host-only validation works, and the product path
refuses to run without a CUDA device (no CPU fallback).  No compute calls."""
from __future__ import annotations

import ctypes as C
import dataclasses
import os
import re

import numpy as np
import pytest

import paper_2607_06337_b200 as ob
from workloads import binary_tree_config1, config_params

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "orchard.h")


def _declared_symbols():
    txt = open(HEADER).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(ob_[a-z0-9_]+)\s*\(", txt)))


def test_library_exports_every_declared_symbol():
    L = ob.load_library()
    names = _declared_symbols()
    assert len(names) >= 18
    for n in names:
        assert hasattr(L, n), f"{n} declared in include/orchard.h but not exported by libob.so"
    assert sorted(ob.EXPORTS) == names


def test_struct_layouts_match_the_header():
    # ob_event: 4 x int32 + 2 x float; ob_params: counted from the header's field list
    assert C.sizeof(ob.ob_event) == 24
    assert C.sizeof(ob.ob_params) == 4 * (1 + 3 + 1 + 1 + 1 + 1 + 1 + 1 + 1 + 1 + 1 + 1 + 1 + 1 + 1 + 1 + 10 + 1 + 8)
    assert C.sizeof(ob.ob_geometry_ranges) == 64
    assert C.sizeof(ob.ob_world_spec) == 8 * 15 if C.sizeof(C.c_void_p) == 8 else True
    L = ob.load_library()
    assert L.ob_sizeof_params() == C.sizeof(ob.ob_params)
    assert L.ob_sizeof_world_spec() == C.sizeof(ob.ob_world_spec)
    assert L.ob_sizeof_event() == C.sizeof(ob.ob_event)


def test_default_params_are_the_documented_readings():
    p = ob.default_params()
    assert abs(p.h - 2e-3) < 1e-9 and tuple(p.gravity) == (0.0, 0.0, np.float32(-9.81))
    assert abs(p.c_d - 0.05) < 1e-8 and abs(p.cg_tol - 1e-6) < 1e-12 and p.cg_max_iter == 200 and p.precond == 2
    assert p.rupture_frames == 3 and p.detach_frames_pull == 3 and p.detach_frames_tension == 10
    assert abs(p.detach_kappa - 1.1) < 1e-6 and p.react_max == 40.0 and p.tether_implicit == 1
    assert p.qd_max == 50.0 and abs(p.zeta_s - 0.1) < 1e-7 and p.forces_off_on_snapped == 1 and p.mass_damping == 0.0
    assert p.fric_frac == 0.0 and p.fric_ramp == 5.0 and p.fric_time == 1.5 and p.snap_drag_scale == 1.0
    assert p.rail_speed == 0.0 and p.rail_fade == 0.5 and p.rail_brake == 50.0
    assert ob.load_library().ob_default_params(None) == ob.OB_E_ARG


def _ws_bytes(specs, params):
    L = ob.load_library()
    arr, keep = ob.marshal_specs(specs)
    n = C.c_size_t(0)
    rc = L.ob_workspace_bytes(arr, len(specs), C.byref(ob.params_struct(params)), C.byref(n))
    return rc, n.value, L.ob_last_error(None).decode()


def test_workspace_bytes_validates_on_the_host():
    spec, P = binary_tree_config1(), config_params(1)
    rc, n, _ = _ws_bytes([spec], P)
    assert rc == ob.OB_OK and n > 0 and n % 256 == 0
    rc2, n2, _ = _ws_bytes([spec, spec], P)
    assert rc2 == ob.OB_OK and n2 > n
    # non-topological parent
    bad = dataclasses.replace(spec, parent=spec.parent.copy())
    bad.parent[3] = 7
    rc, _, msg = _ws_bytes([bad], P)
    assert rc == ob.OB_E_ARG and "topological" in msg
    # non-unit quaternion
    bad = dataclasses.replace(spec, rest_quat=spec.rest_quat.copy())
    bad.rest_quat[5] *= 1.01
    assert _ws_bytes([bad], P)[0] == ob.OB_E_ARG
    # non-positive diameter, apple on a link that does not exist
    bad = dataclasses.replace(spec, diameter=spec.diameter.copy())
    bad.diameter[2] = 0.0
    assert _ws_bytes([bad], P)[0] == ob.OB_E_ARG
    bad = dataclasses.replace(spec, apple_link=np.array([15, 19, 23, 31], dtype=np.int32))
    assert _ws_bytes([bad], P)[0] == ob.OB_E_ARG
    # bad params
    assert _ws_bytes([spec], dataclasses.replace(P, h=0.0))[0] == ob.OB_E_ARG
    assert _ws_bytes([spec], dataclasses.replace(P, rupture_frames=0))[0] == ob.OB_E_ARG
    # empty batch
    L = ob.load_library()
    n = C.c_size_t(0)
    assert L.ob_workspace_bytes(None, 0, C.byref(ob.params_struct(P)), C.byref(n)) == ob.OB_E_ARG


def test_capacity_limits_are_reported_not_crashed():
    """A link with more children than the packed topology word holds (15), or a world too large for one CTA's
    shared memory, is refused with OB_E_CAPACITY by the host-side planner."""
    P = config_params(1)
    n = 18
    star = ob_star_spec(n)
    rc, _, msg = _ws_bytes([star], P)
    assert rc == ob.OB_E_CAPACITY and "children" in msg
    rc, _, _ = _ws_bytes([ob_star_spec(16)], P)          # 15 children: fine
    assert rc == ob.OB_OK
    # the largest worlds of BASELINE.json configs[4] (1500 links, 150 apples) must fit into one CTA's shared memory
    from workloads import stochastic_world
    big = stochastic_world(np.random.default_rng(3), 1497, 1500, 150, depth_choices=(7, 8))
    assert big.n_links >= 1497 and _ws_bytes([big], config_params(5))[0] == ob.OB_OK


def ob_star_spec(n_links):
    from workloads import WorldSpec
    q = np.zeros((n_links, 4), np.float32)
    q[:, 0] = 1.0
    return WorldSpec(parent=np.array([-1] + [0] * (n_links - 1), np.int32), length=np.full(n_links, 0.3, np.float32),
                     diameter=np.full(n_links, 0.02, np.float32), rest_quat=q, density=800.0, E=8e9, MOR=6e7,
                     apple_link=np.zeros(0, np.int32), apple_offset=np.zeros((0, 3), np.float32),
                     apple_mass=np.zeros(0, np.float32), apple_radius=np.zeros(0, np.float32),
                     apple_k=np.zeros(0, np.float32), apple_c=None, apple_detach=np.zeros(0, np.float32))


def test_null_context_calls_return_arg_errors():
    L = ob.load_library()
    assert L.ob_step(None, 1) == ob.OB_E_ARG
    assert L.ob_randomize(None, 1) == ob.OB_E_ARG
    n = C.c_int(0)
    assert L.ob_events(None, None, 0, C.byref(n)) == ob.OB_E_ARG
    assert L.ob_stats(None, None, None, None) == ob.OB_E_ARG
    assert isinstance(L.ob_last_error(None), bytes)
    L.ob_destroy(None)   # no-op


def test_no_cpu_fallback():
    """Without a CUDA device ob_create returns OB_E_CUDA and the binding raises; nothing routes to oracle/."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    spec, P = binary_tree_config1(), config_params(1)
    L = ob.load_library()
    arr, keep = ob.marshal_specs([spec])
    ps = ob.params_struct(P)
    n = C.c_size_t(0)
    assert L.ob_workspace_bytes(arr, 1, C.byref(ps), C.byref(n)) == ob.OB_OK
    h = C.c_void_p()
    rc = L.ob_create(arr, 1, C.byref(ps), C.c_void_p(256), n, None, C.byref(h))
    assert rc == ob.OB_E_CUDA and not h.value
    with pytest.raises(RuntimeError):
        ob.Orchard([spec], P)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2607_06337_b200")
    for dirpath, _dirs, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "orchard_oracle" not in src, f
    for dirpath, _dirs, files in os.walk(os.path.join(ROOT, "oracle")):
        for f in files:
            if f.endswith((".py", ".c", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import paper_2607_06337_b200" not in src and "libob" not in src, f
