"""-m "not gpu": the C-ABI library builds for sm_100a, loads without a GPU and exports every symbol that
include/emx.h declares; argument checks that need no device behave as documented."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    from paper_2203_09467_b200 import build, emx
    build.build()
    return emx.lib()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "emx.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(emx_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(L):
    from paper_2203_09467_b200 import emx
    names = declared_symbols()
    assert len(names) >= 25
    for n in names:
        assert hasattr(L, n), n
    assert sorted(emx.EXPORTS) == names


def test_struct_layouts_match_the_header(L):
    from paper_2203_09467_b200 import emx
    from oracle import emo
    assert C.sizeof(emx.Track) == 88 and C.sizeof(emx.Track) == C.sizeof(emo.Track)
    assert C.sizeof(emx.StepResult) == C.sizeof(emo.StepResult)
    assert C.sizeof(emx.Physics) == C.sizeof(emo.Physics)


def test_host_side_argument_checks_without_a_device(L):
    h = C.c_void_p()
    assert L.emx_create(C.byref(h)) == 0
    Z = (C.c_int * 1)(82); A = (C.c_double * 1)(207.2); w = (C.c_double * 1)(1.0)
    assert L.emx_add_material(h, 1, Z, A, w, 11.35, 823.0) == 0
    assert L.emx_add_material(h, 0, Z, A, w, 11.35, 823.0) == -1
    assert L.emx_add_material(h, 1, Z, A, w, -1.0, 823.0) == -1
    assert L.emx_add_surface(h, 2, 0.0) == 0 and L.emx_add_surface(h, 2, 1.0) == 1
    assert L.emx_add_surface(h, 3, -5.0) == -1 and L.emx_add_surface(h, 7, 1.0) == -1
    s = (C.c_int * 2)(0, 1); e = (C.c_int * 2)(1, -1)
    assert L.emx_add_volume(h, 2, s, e, 0, 0) == 0
    assert L.emx_add_volume(h, 2, s, e, 5, 0) == -1          # unknown material
    bad = (C.c_int * 2)(0, 9)
    assert L.emx_add_volume(h, 2, bad, e, 0, 0) == -1        # unknown surface
    assert L.emx_n_tally(h) == 1
    from paper_2203_09467_b200 import emx
    ph = emx.Physics()
    assert L.emx_get_physics(h, C.byref(ph)) == 0
    assert (ph.n_E, ph.alpha_R, ph.rho_R, ph.max_steps) == (256, 0.2, 0.1, 10000)
    ph.n_E = 1
    assert L.emx_set_physics(h, C.byref(ph)) == -1
    assert L.emx_workspace_bytes(h, 1 << 20, 1 << 26) > (1 << 20) * 84 + (1 << 26) * 80 * 0.9
    assert L.emx_workspace_bytes(h, 0, 10) == 0 and L.emx_workspace_bytes(h, (1 << 22) + 1, 10) == 0
    L.emx_staging_bytes.restype, L.emx_staging_bytes.argtypes = C.c_size_t, [C.c_long]
    assert L.emx_staging_bytes(100000) >= 100000 * 68 and L.emx_staging_bytes(0) > 0
    # the schedule: defaults, validation (it never changes a result, so there is nothing else to check without a GPU)
    sc = emx.Schedule()
    assert L.emx_get_schedule(h, C.byref(sc)) == 0
    assert (sc.loop_node, sc.slice_min, sc.slice_above) == (1, 2, -1) and sc.slice_max >= sc.slice_min
    sc.slice_min = 0
    assert L.emx_set_schedule(h, C.byref(sc)) == -1
    sc.slice_min, sc.slice_max = 4, 3
    assert L.emx_set_schedule(h, C.byref(sc)) == -1
    sc.slice_max = 8
    sc.blocks_per_sm[3] = 17
    assert L.emx_set_schedule(h, C.byref(sc)) == -1
    sc.blocks_per_sm[3] = 4
    assert L.emx_set_schedule(h, C.byref(sc)) == 0
    sc2 = emx.Schedule()
    assert L.emx_get_schedule(h, C.byref(sc2)) == 0 and (sc2.slice_min, sc2.slice_max, sc2.blocks_per_sm[3]) == (4, 8, 4)
    # compute calls before the tables are built are refused with EMX_E_STATE
    assert L.emx_read_tallies(h, None, None) == -2
    assert L.emx_step_batch(h, 0, 0, None, None, None) == -2
    assert b"not built" in L.emx_last_error(h)
    L.emx_destroy(h)
    assert L.emx_version().startswith(b"emx")


def test_no_cpu_fallback_without_a_device(L):
    """On a box with no GPU the product path must fail loudly, not compute on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2203_09467_b200 import emx, workloads as W
    desc, _ = W.config0(4)
    with pytest.raises(RuntimeError):
        emx.Problem(desc)
    P = emx.Problem(desc, build=False)
    assert L.emx_build_tables(P.h, None) == -3               # EMX_E_CUDA
