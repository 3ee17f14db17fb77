"""CPU tests of the C-ABI boundary and its host logic: the library loads without a GPU, exports
every symbol include/sph.h declares, and its host-side geometry / sizing agree with the oracle's
independent statement of reading R11."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_2403_11156_b200 import scenes

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def binding():
    from paper_2403_11156_b200 import binding, build
    build.build()
    return binding


def declared_functions():
    src = open(os.path.join(ROOT, "include", "sph.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sph_[a-z_]+)\s*\(", src)))


def test_library_loads_and_exports_every_declared_symbol(binding):
    lib = binding.load()
    names = declared_functions()
    assert len(names) >= 12
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(binding.EXPORTS) == names


def test_struct_sizes_match_header(binding):
    """ctypes mirrors of the C structs: field counts of the header and sizes."""
    src = open(os.path.join(ROOT, "include", "sph.h")).read()
    body = re.search(r"typedef struct SphParams \{(.*?)\} SphParams;", src, re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    n_scalars = 0
    for decl in body.split(";"):
        decl = decl.strip()
        if not decl:
            continue
        names = decl.split(None, 1)[1].split(",")
        for nm in names:
            m = re.search(r"\[(\d+)\]", nm)
            n_scalars += int(m.group(1)) if m else 1
    assert ctypes.sizeof(binding.SphParams) == 4 * n_scalars
    assert ctypes.sizeof(binding.SphRigidBody) == 4 * 21
    assert ctypes.sizeof(binding.SphBuffers) == 6 * 8


@pytest.mark.parametrize("idx", [0, 1, 2, 3, 4])
def test_grid_geometry_matches_oracle_for_every_config(binding, oracle, idx):
    """Host logic (R11): n_a = floor((max - o) / c) + 1 with fp32 c = h (1 + 2^-10)."""
    if idx == 0:
        sc = scenes.config(0)
    else:  # geometry only depends on the parameters: shrink the particle arrays
        sc = scenes.config(idx)
    p = binding.make_params(sc.params)
    (nx, ny, nz, nc), (kf, kb) = binding.sph_grid_dims(p)
    tiny = oracle.Sim(sc.fluid_pos[:1], sc.fluid_vel[:1], np.zeros((0, 3), np.float32), np.zeros(0, np.int32), [], sc.params)
    tiny.build_grid()
    assert (nx, ny, nz, nc) == tuple(tiny.grid_dims(0))
    assert kf == 64 and kb == 64
    need = binding.sph_workspace_bytes(p, sc.n_fluid, sc.n_boundary, len(sc.bodies))
    # SoA store + lists: a few hundred bytes per particle, never absurd
    assert 200 * sc.n_fluid < need < 2000 * (sc.n_fluid + sc.n_boundary) + 64 * nc + (1 << 20)


def test_invalid_parameters_are_rejected_without_a_gpu(binding):
    sc = scenes.config(0)
    prm = dict(sc.params)
    prm["support_radius"] = 0.0
    assert binding.sph_workspace_bytes(binding.make_params(prm), 10, 0, 0) == 0
    prm = dict(sc.params)
    prm["domain_max"] = (1e9, 1e9, 1e9)
    assert binding.sph_workspace_bytes(binding.make_params(prm), 10, 0, 0) == 0
    with pytest.raises(binding.SphError):
        binding.sph_grid_dims(binding.make_params(prm))
    p = binding.make_params(dict(sc.params, max_fluid_neighbors=30, max_boundary_neighbors=7))
    assert binding.sph_grid_dims(p)[1] == (32, 8)


def test_product_path_has_no_cpu_fallback(binding):
    import torch
    if torch.cuda.is_available():
        pytest.skip("CPU-only check")
    sc = scenes.dam_break((4, 4, 4), (6, 6, 6))
    with pytest.raises(RuntimeError):
        binding.Sim.from_scene(sc)


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2403_11156_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "sphref" not in txt and "import oracle" not in txt and "from oracle" not in txt, f


def test_round2_host_logic_without_a_gpu(binding):
    """Host-side argument checks and sizing of the round-2 entry points (no compute call is made):
    warm-start factor range, surface-grid sizing, NULL / size rejection of the selection and slab calls."""
    sc = scenes.config(0)
    assert binding.sph_workspace_bytes(binding.make_params(dict(sc.params, warm_start=1, warm_start_factor=1.5)), 10, 0, 0) == 0
    cold = binding.sph_workspace_bytes(binding.make_params(sc.params), 1000, 0, 0)
    warm = binding.sph_workspace_bytes(binding.make_params(dict(sc.params, warm_start=1)), 1000, 0, 0)
    assert warm >= cold + 2 * 4 * 1000                     # the two running-total arrays
    L = binding.load()
    sp = binding.SphSurfaceParams()
    sp.grid_min = (ctypes.c_float * 3)(0, 0, 0); sp.cube_size = 0.01; sp.iso = 0.6
    sp.dims = (ctypes.c_int * 3)(10, 20, 30)
    need = L.sph_surface_workspace_bytes(ctypes.byref(sp))
    assert 4 * 6000 + 4 * 9 * 19 * 29 <= need <= 4 * 6000 + 4 * 9 * 19 * 29 + 4096
    sp.dims = (ctypes.c_int * 3)(1, 20, 30)                 # fewer than 2 nodes on an axis: no cells
    assert L.sph_surface_workspace_bytes(ctypes.byref(sp)) == 0
    sp.dims = (ctypes.c_int * 3)(10, 20, 30); sp.cube_size = 0.0
    assert L.sph_surface_workspace_bytes(ctypes.byref(sp)) == 0
    cnt = ctypes.c_int(7)
    assert L.sph_select_range(None, None, None, None, None, 0, 5, 0.0, 1.0, None, None, None, None, 0, None, 0,
                              ctypes.byref(cnt)) == binding.SPH_EINVAL      # no scratch
    assert L.sph_slab_phase(None, 0) == binding.SPH_EINVAL
    assert L.sph_surface_extract(None, ctypes.byref(sp), None, 0, None, 0, None) == binding.SPH_EINVAL
    assert L.sph_step_pcisph(None, 1) == binding.SPH_EINVAL
