"""No-GPU checks of the boundary: libcfneb.so builds for sm_100a, loads, and exports every symbol include/cfneb.h
declares; the calls that need no device behave as the header says; the product path has no CPU fallback and never
touches oracle/; the seeded workload generators give the shapes of BASELINE.json's configs."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def cf():
    import paper_2510_16721_b200 as cf
    from paper_2510_16721_b200 import build
    build.build()  # nvcc cross-compiles without a GPU; no-op when the library is newer than its sources
    return cf


def header_symbols():
    text = open(os.path.join(ROOT, "include", "cfneb.h")).read()
    return sorted(set(re.findall(r"CFNEB_API\s+[\w\s\*]+?\b(cfneb_\w+)\s*\(", text)))


def test_library_exports_every_declared_symbol(cf):
    names = header_symbols()
    assert len(names) >= 20 and "cfneb_create" in names and "cfneb_step" in names
    L = ctypes.CDLL(cf.LIB_PATH)
    for n in names:
        assert getattr(L, n) is not None, n
    assert sorted(cf.EXPORTS) == names  # the binding wraps exactly the header's entry points


def test_params_struct_layout_and_defaults(cf):
    assert ctypes.sizeof(cf.Params) == 8 * 4 + (12 + 2 + 7 + 1 + 1) * 8 + 8   # ... + the types pointer
    p = cf.default_params()
    assert (p.potential, p.cell_mode, p.climb, p.fire_nmin) == (cf.POT_LJ_SF, cf.CELL_B, 1, 5)
    assert (p.fire_dt0, p.fire_dtmax, p.fire_maxstep, p.fire_finc, p.fire_fdec, p.fire_astart, p.fire_fa) == (
        0.1, 1.0, 0.2, 1.1, 0.5, 0.1, 0.99)
    assert p.skin == 0.3 and p.pressure == 0.0 and p.k_spring == 1.0 and p.cell_factor == 1.0
    assert list(p.pot)[:3] == [1.0, 1.0, 2.5]
    with pytest.raises(KeyError):
        cf.default_params(no_such_field=1)


def test_workspace_bytes_and_argument_errors_need_no_device(cf):
    from cfneb_workloads import CONFIGS
    prm = cf.params_for(CONFIGS[4], cell_factor=0.0)
    ws = cf.workspace_bytes(CONFIGS[4].n_atoms, prm)
    state = 72 * CONFIGS[4].n_atoms * 100            # X (x2 buffers aside), v, F of 100 images
    lists = 4 * 224 * CONFIGS[4].n_atoms * 100       # the uint32 lists at the config's capacity
    assert 2 * state + lists < ws < 14e9             # no scratch of the size of the lists (round 1: 23.6 GB)
    assert cf.workspace_bytes(0, prm) == 0           # invalid n_atoms
    bad = cf.params_for(CONFIGS[4], cell_factor=0.0)
    bad.max_images = 2
    assert cf.workspace_bytes(100, bad) == 0
    L = cf.lib()
    out = ctypes.c_void_p()
    assert L.cfneb_create(ctypes.byref(out), 10, None, None, None, None, 5, None, ctypes.byref(prm), None, 0, None) == -1
    assert out.value is None
    assert L.cfneb_step(None, 1) == -1 and L.cfneb_get_status(None, None) == -1
    assert L.cfneb_relax_endpoints(None, 1e-3, 10, 1, None, None, None) == -1
    assert L.cfneb_step_adaptive(None, 1, 1, 1.0, 0.1) == -1
    assert L.cfneb_get_checkpoint(None, None, None, None, None, None) == -1
    assert L.cfneb_set_state(None, None, None, None, None, None) == -1
    assert L.cfneb_step_hosted(None, None, None, None, 0) == -1 and L.cfneb_reparametrize(None, 1) == -1
    assert ctypes.sizeof(cf.FireState) == 32
    assert L.cfneb_get_dots(None, None, None, None) == -1
    # the no-allocation entry point checks its sizes before it touches the device
    assert L.cfneb_band_dots_noalloc(None, None, None, 2, 10, None, None) == -1
    assert L.cfneb_band_dots_noalloc(None, None, None, cf.NOALLOC_MAX_IMAGES + 1, 10, None, None) == -7
    assert b"CFNEB_NOALLOC_MAX_IMAGES = 128" in L.cfneb_band_dots_noalloc_error()
    assert re.search(r"#define\s+CFNEB_NOALLOC_MAX_IMAGES\s+128\b", open(os.path.join(ROOT, "include", "cfneb.h")).read())
    for code in range(0, -8, -1):
        assert len(L.cfneb_strerror(code)) > 1
    L.cfneb_destroy(None)  # documented no-op


def test_no_cpu_fallback_and_no_oracle_in_the_product(cf):
    import torch
    pkg = os.path.join(ROOT, "paper_2510_16721_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, re.M), f
                assert "liboracle" not in text, f
    if not torch.cuda.is_available():
        from cfneb_workloads import build_workload
        spec, pos, cells = build_workload(0)
        with pytest.raises(Exception):  # no device: the binding refuses, it does not compute on the host
            cf.CFNEB(pos, cells, cf.params_for(spec))


def test_workload_generators_match_baseline_configs():
    from cfneb_workloads import CONFIGS, build_workload, splitmix64_normals
    shapes = {0: (7, 31), 1: (9, 255), 2: (16, 2048)}
    for k, (P, N) in shapes.items():
        spec, pos, cells = build_workload(k)
        assert pos.shape == (P, N, 3) and cells.shape == (P, 3, 3)
        assert (spec.n_images, spec.n_atoms) == (P, N)
        spec2, pos2, cells2 = build_workload(k)
        assert np.array_equal(pos, pos2) and np.array_equal(cells, cells2)      # seeded
        assert np.all(np.linalg.det(cells) > 0)
    assert (CONFIGS[3].n_atoms, CONFIGS[3].n_images) == (9826, 12)
    assert (CONFIGS[4].n_atoms, CONFIGS[4].n_images) == (101306, 100)
    z = splitmix64_normals(7, 20000)
    assert np.array_equal(z, splitmix64_normals(7, 20000)) and not np.array_equal(z, splitmix64_normals(8, 20000))
    assert abs(z.mean()) < 0.03 and abs(z.std() - 1.0) < 0.03
    # interior images carry the noise, endpoints do not (Bain: endpoints are perfect lattices)
    spec, pos, cells = build_workload(2, 4, dims=(3, 3, 3))
    frac0 = pos[0] @ np.linalg.inv(cells[0])
    assert np.max(np.abs(frac0 * 6 - np.round(frac0 * 6))) < 1e-9
    frac1 = pos[1] @ np.linalg.inv(cells[1])
    assert 1e-5 < np.max(np.abs(frac1 * 6 - np.round(frac1 * 6))) < 1e-2
