"""Thin ctypes binding of libsph_b200.so (include/sph.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; this module converts
dictionaries / dataclasses to the C structs, hands over raw device pointers of PyTorch
tensors (PyTorch only holds the device memory and the stream) and returns tensors.
There is NO CPU fallback: if the library has not been built (python -m
paper_2403_11156_b200.build) loading raises, and creating a simulation without a CUDA
device raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, Optional, Sequence

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsph_b200.so")

SPH_OK, SPH_EINVAL, SPH_ENOMEM, SPH_ECUDA, SPH_EDOMAIN, SPH_ESTATE = 0, -1, -2, -3, -4, -5

# SphField
(POS, VEL, DENSITY, ALPHA, KAPPA_OVER_RHO, CELL_START, CELL_OF_PARTICLE, SORTED_ID, NEIGHBOR_COUNT,
 FLUID_NEIGHBORS, BOUNDARY_NEIGHBORS, BOUNDARY_POS, BOUNDARY_VEL, BOUNDARY_PSI, BOUNDARY_FORCE,
 RIGID_BODIES, BOUNDARY_CELL_START, BOUNDARY_CELL_OF_PARTICLE, KSUM_DIVERGENCE, KSUM_DENSITY) = range(20)

EXPORTS = ["sph_workspace_bytes", "sph_grid_dims", "sph_create", "sph_build_grid", "sph_step_dfsph",
           "sph_step_wcsph", "sph_step_pcisph", "sph_set_forced_iterations", "sph_read_state", "sph_write_state",
           "sph_read_stats", "sph_host_sync", "sph_launch_count", "sph_enable_kernel_timing", "sph_read_kernel_times",
           "sph_surface_workspace_bytes", "sph_surface_extract", "sph_slab_set_particles", "sph_slab_phase",
           "sph_slab_gather", "sph_slab_scatter", "sph_slab_read_error_sum", "sph_slab_set_loop", "sph_slab_store",
           "sph_select_range", "sph_select_range_static", "sph_render_workspace_bytes", "sph_render_particles",
           "sph_last_error", "sph_destroy"]


class SphParams(C.Structure):
    _fields_ = [
        ("particle_radius", C.c_float), ("support_radius", C.c_float), ("rest_density", C.c_float),
        ("particle_mass", C.c_float), ("dt", C.c_float), ("gravity", C.c_float * 3),
        ("domain_min", C.c_float * 3), ("domain_max", C.c_float * 3),
        ("tank_min", C.c_float * 3), ("tank_max", C.c_float * 3),
        ("viscosity_mode", C.c_int), ("kinematic_viscosity", C.c_float),
        ("cg_rel_tol", C.c_float), ("cg_max_iter", C.c_int),
        ("eta_density", C.c_float), ("min_iter_density", C.c_int), ("max_iter_density", C.c_int),
        ("eta_divergence", C.c_float), ("min_iter_divergence", C.c_int), ("max_iter_divergence", C.c_int),
        ("enable_divergence_solve", C.c_int), ("force_iterations", C.c_int),
        ("wcsph_stiffness", C.c_float), ("wcsph_exponent", C.c_float),
        ("max_fluid_neighbors", C.c_int), ("max_boundary_neighbors", C.c_int),
        ("use_cuda_graph", C.c_int), ("use_neighbor_list", C.c_int),
        ("cfl_factor", C.c_float), ("dt_min", C.c_float),
        ("warm_start", C.c_int), ("warm_start_factor", C.c_float),
        ("pcisph_min_iter", C.c_int), ("pcisph_max_iter", C.c_int),
    ]


class SphRigidBody(C.Structure):
    _fields_ = [
        ("first_particle", C.c_int), ("n_particles", C.c_int), ("dynamic", C.c_int),
        ("mass", C.c_float), ("inertia_body", C.c_float * 3), ("com", C.c_float * 3),
        ("quat", C.c_float * 4), ("lin_vel", C.c_float * 3), ("ang_vel", C.c_float * 3),
        ("contact_radius", C.c_float),
    ]


class SphBuffers(C.Structure):
    _fields_ = [
        ("fluid_pos", C.c_void_p), ("fluid_vel", C.c_void_p), ("boundary_pos", C.c_void_p),
        ("boundary_body", C.c_void_p), ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t),
    ]


class SphStats(C.Structure):
    _fields_ = [
        ("steps_done", C.c_longlong), ("total_it_v", C.c_longlong), ("total_it_d", C.c_longlong),
        ("total_cg_iters", C.c_longlong),
        ("it_v", C.c_int), ("it_d", C.c_int), ("cg_iters", C.c_int),
        ("err_v", C.c_float), ("err_rho", C.c_float), ("cg_residual", C.c_float),
        ("oob_count", C.c_int), ("overflow_count", C.c_int), ("nan_count", C.c_int),
        ("max_iter_hit", C.c_int), ("v_max", C.c_float),
        ("max_fluid_neighbors", C.c_int), ("max_boundary_neighbors", C.c_int),
        ("mean_fluid_neighbors", C.c_float), ("dt_last", C.c_float), ("sim_time", C.c_double),
    ]


class SphSurfaceParams(C.Structure):
    _fields_ = [("grid_min", C.c_float * 3), ("dims", C.c_int * 3), ("cube_size", C.c_float), ("iso", C.c_float)]


class SphRenderParams(C.Structure):
    _fields_ = [("origin", C.c_float * 3), ("right", C.c_float * 3), ("up", C.c_float * 3), ("pixel_size", C.c_float),
                ("width", C.c_int), ("height", C.c_int), ("radius", C.c_float), ("light", C.c_float * 3)]


class SphError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"libsph_b200 error {code}: {text}")
        self.code = code


_lib = None


def load() -> C.CDLL:
    """dlopen the C-ABI library; raises if it has not been built (no fallback of any kind)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(
                f"{LIB_PATH} is missing: build the CUDA library first "
                "(python -m paper_2403_11156_b200.build); there is no CPU fallback")
        L = C.CDLL(LIB_PATH)
        pp = C.POINTER(SphParams)
        L.sph_workspace_bytes.restype = C.c_size_t
        L.sph_workspace_bytes.argtypes = [pp, C.c_int, C.c_int, C.c_int]
        L.sph_grid_dims.argtypes = [pp, C.POINTER(C.c_int), C.POINTER(C.c_int)]
        L.sph_create.argtypes = [pp, C.POINTER(SphBuffers), C.c_int, C.c_int, C.POINTER(SphRigidBody),
                                 C.c_int, C.c_int, C.c_void_p, C.POINTER(C.c_void_p)]
        L.sph_build_grid.argtypes = [C.c_void_p]
        L.sph_step_dfsph.argtypes = [C.c_void_p, C.c_int]
        L.sph_step_wcsph.argtypes = [C.c_void_p, C.c_int]
        L.sph_step_pcisph.argtypes = [C.c_void_p, C.c_int]
        L.sph_set_forced_iterations.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int]
        L.sph_read_state.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_size_t, C.c_int]
        L.sph_write_state.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_size_t, C.c_int]
        L.sph_read_stats.argtypes = [C.c_void_p, C.POINTER(SphStats)]
        L.sph_host_sync.argtypes = [C.c_void_p]
        L.sph_launch_count.restype = C.c_longlong
        L.sph_launch_count.argtypes = [C.c_void_p]
        L.sph_enable_kernel_timing.argtypes = [C.c_void_p, C.c_int]
        L.sph_read_kernel_times.argtypes = [C.c_void_p, C.c_char_p, C.c_size_t]
        L.sph_surface_workspace_bytes.restype = C.c_size_t
        L.sph_surface_workspace_bytes.argtypes = [C.POINTER(SphSurfaceParams)]
        L.sph_surface_extract.argtypes = [C.c_void_p, C.POINTER(SphSurfaceParams), C.c_void_p, C.c_size_t, C.c_void_p,
                                          C.c_longlong, C.POINTER(C.c_longlong)]
        L.sph_slab_set_particles.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int]
        L.sph_slab_phase.argtypes = [C.c_void_p, C.c_int]
        L.sph_slab_gather.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.c_void_p]
        L.sph_slab_scatter.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p]
        L.sph_slab_read_error_sum.argtypes = [C.c_void_p, C.POINTER(C.c_ulonglong)]
        L.sph_slab_set_loop.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_float]
        L.sph_slab_store.argtypes = [C.c_void_p, C.POINTER(C.c_void_p), C.POINTER(C.c_void_p), C.POINTER(C.c_void_p),
                                     C.POINTER(C.c_int), C.POINTER(C.c_int)]
        L.sph_select_range.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int,
                                       C.c_float, C.c_float, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int,
                                       C.c_void_p, C.c_size_t, C.POINTER(C.c_int)]
        L.sph_select_range_static.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int,
                                              C.c_float, C.c_float, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int,
                                              C.POINTER(C.c_int)]
        L.sph_render_workspace_bytes.restype = C.c_size_t
        L.sph_render_workspace_bytes.argtypes = [C.POINTER(SphRenderParams), C.c_int]
        L.sph_render_particles.argtypes = [C.c_void_p, C.POINTER(SphRenderParams), C.c_void_p, C.c_size_t,
                                           C.c_void_p, C.c_void_p, C.c_void_p]
        L.sph_last_error.restype = C.c_char_p
        L.sph_last_error.argtypes = [C.c_void_p]
        L.sph_destroy.argtypes = [C.c_void_p]
        L.sph_destroy.restype = None
        _lib = L
    return _lib


def make_params(prm: Dict[str, object]) -> SphParams:
    """dict (keys of scenes.default_params + optional library switches) -> SphParams."""
    p = SphParams()
    defaults = dict(max_fluid_neighbors=0, max_boundary_neighbors=0, use_cuda_graph=1, use_neighbor_list=1,
                    cfl_factor=0.0, dt_min=0.0, warm_start=0, warm_start_factor=0.5, pcisph_min_iter=0, pcisph_max_iter=0)
    for name, ctype in SphParams._fields_:
        val = prm.get(name, defaults.get(name))
        if val is None:
            raise KeyError(f"parameter {name} missing")
        if hasattr(ctype, "_length_"):
            setattr(p, name, ctype(*[float(v) for v in val]))
        else:
            setattr(p, name, val)
    return p


def make_bodies(bodies: Sequence[object]):
    arr = (SphRigidBody * max(1, len(bodies)))()
    for i, b in enumerate(bodies):
        g = (lambda k: b[k]) if isinstance(b, dict) else (lambda k: getattr(b, k))
        arr[i].first_particle = int(g("first_particle"))
        arr[i].n_particles = int(g("n_particles"))
        arr[i].dynamic = int(g("dynamic"))
        arr[i].mass = float(g("mass"))
        arr[i].inertia_body = (C.c_float * 3)(*[float(v) for v in g("inertia_body")])
        arr[i].com = (C.c_float * 3)(*[float(v) for v in g("com")])
        arr[i].quat = (C.c_float * 4)(*[float(v) for v in g("quat")])
        arr[i].lin_vel = (C.c_float * 3)(*[float(v) for v in g("lin_vel")])
        arr[i].ang_vel = (C.c_float * 3)(*[float(v) for v in g("ang_vel")])
        arr[i].contact_radius = float(g("contact_radius"))
    return arr


def sph_workspace_bytes(params: SphParams, n_fluid: int, n_boundary: int, n_bodies: int) -> int:
    return int(load().sph_workspace_bytes(C.byref(params), n_fluid, n_boundary, n_bodies))


def sph_grid_dims(params: SphParams):
    d = (C.c_int * 4)()
    k = (C.c_int * 2)()
    rc = load().sph_grid_dims(C.byref(params), d, k)
    if rc != SPH_OK:
        raise SphError(rc, "sph_grid_dims")
    return tuple(d[:]), tuple(k[:])


class Sim:
    """One simulation handle.  Owns the PyTorch tensors that back the workspace."""

    def __init__(self, fluid_pos, fluid_vel, boundary_pos, boundary_body, bodies, params: Dict[str, object],
                 device: int = 0, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("libsph_b200 needs a CUDA device; there is no CPU fallback")
        L = load()
        self._torch = torch
        self.device = torch.device("cuda", device)
        self.params = make_params(params)
        self.nf = int(len(fluid_pos))
        self.nb = int(len(boundary_pos)) if boundary_pos is not None else 0
        self.nbodies = len(bodies)
        self._bodies = make_bodies(bodies)
        (self.nx, self.ny, self.nz, self.ncells), (self.kf, self.kb) = sph_grid_dims(self.params)
        f32, i32 = torch.float32, torch.int32
        dev = self.device
        as_dev = lambda a, dt: torch.as_tensor(a, dtype=dt).contiguous().to(dev)
        self._in = [as_dev(fluid_pos, f32).reshape(-1), as_dev(fluid_vel, f32).reshape(-1)]
        if self.nb:
            self._in += [as_dev(boundary_pos, f32).reshape(-1), as_dev(boundary_body, i32).reshape(-1)]
        nbytes = sph_workspace_bytes(self.params, self.nf, self.nb, self.nbodies)
        if nbytes == 0:
            raise SphError(SPH_EINVAL, "sph_workspace_bytes rejected the parameters")
        self.workspace_bytes = nbytes
        self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=dev)
        base = self._ws.data_ptr()
        aligned = (base + 255) & ~255
        buf = SphBuffers()
        buf.fluid_pos = self._in[0].data_ptr() if self.nf else None
        buf.fluid_vel = self._in[1].data_ptr() if self.nf else None
        buf.boundary_pos = self._in[2].data_ptr() if self.nb else None
        buf.boundary_body = self._in[3].data_ptr() if self.nb else None
        buf.workspace = aligned
        buf.workspace_bytes = nbytes
        # own stream: a CUDA graph cannot be captured on the legacy default stream
        self._stream = stream if stream is not None else torch.cuda.Stream(dev)
        self._stream.wait_stream(torch.cuda.current_stream(dev))   # inputs were staged by torch
        h = C.c_void_p()
        rc = L.sph_create(C.byref(self.params), C.byref(buf), self.nf, self.nb, self._bodies, self.nbodies,
                          device, C.c_void_p(self._stream.cuda_stream), C.byref(h))
        if rc != SPH_OK:
            raise SphError(rc, (L.sph_last_error(None) or b"").decode())
        self._h = h
        self._in = None   # inputs were copied into the workspace (sph_create synchronised)

    @property
    def stream(self):
        return self._stream

    def _after_read(self, out):
        """Order torch's current stream after the simulation stream for a tensor just written."""
        cur = self._torch.cuda.current_stream(self.device)
        if cur != self._stream:
            out.record_stream(self._stream)
            cur.wait_stream(self._stream)
        return out

    @classmethod
    def from_scene(cls, scene, device: int = 0, **overrides):
        prm = dict(scene.params)
        prm.update(overrides)
        return cls(scene.fluid_pos, scene.fluid_vel, scene.boundary_pos, scene.boundary_body, scene.bodies,
                   prm, device=device)

    # ---- calls (same names as the C ABI)
    def _check(self, rc: int):
        if rc != SPH_OK:
            raise SphError(rc, (load().sph_last_error(self._h) or b"").decode())

    def sph_build_grid(self):
        self._check(load().sph_build_grid(self._h))

    def sph_step_dfsph(self, n_steps: int = 1):
        self._check(load().sph_step_dfsph(self._h, n_steps))

    def sph_step_wcsph(self, n_steps: int = 1):
        self._check(load().sph_step_wcsph(self._h, n_steps))

    def sph_step_pcisph(self, n_steps: int = 1):
        self._check(load().sph_step_pcisph(self._h, n_steps))

    def sph_set_forced_iterations(self, forced_v: int = -1, forced_d: int = -1, forced_cg: int = -1):
        self._check(load().sph_set_forced_iterations(self._h, forced_v, forced_d, forced_cg))

    def _field_shape(self, field: int):
        t = self._torch
        nf, nb = self.nf, self.nb
        table = {
            POS: ((nf, 3), t.float32), VEL: ((nf, 3), t.float32), DENSITY: ((nf,), t.float32),
            ALPHA: ((nf,), t.float32), KAPPA_OVER_RHO: ((nf,), t.float32),
            KSUM_DIVERGENCE: ((nf,), t.float32), KSUM_DENSITY: ((nf,), t.float32),
            CELL_START: ((self.ncells + 1,), t.int32), CELL_OF_PARTICLE: ((nf,), t.int32),
            SORTED_ID: ((nf,), t.int32), NEIGHBOR_COUNT: ((nf, 2), t.int32),
            FLUID_NEIGHBORS: ((nf, self.kf), t.int32), BOUNDARY_NEIGHBORS: ((nf, self.kb), t.int32),
            BOUNDARY_POS: ((nb, 3), t.float32), BOUNDARY_VEL: ((nb, 3), t.float32),
            BOUNDARY_PSI: ((nb,), t.float32), BOUNDARY_FORCE: ((nb, 3), t.float32),
            BOUNDARY_CELL_START: ((self.ncells + 1,), t.int32), BOUNDARY_CELL_OF_PARTICLE: ((nb,), t.int32),
        }
        return table[field]

    def sph_read_state(self, field: int, out=None):
        """Device read: returns a CUDA tensor (asynchronous on the simulation's stream)."""
        t = self._torch
        if field == RIGID_BODIES:
            return self.read_bodies()
        shape, dt = self._field_shape(field)
        if out is None:
            out = t.empty(shape, dtype=dt, device=self.device)
        nbytes = out.numel() * out.element_size()
        self._stream.wait_stream(t.cuda.current_stream(self.device))
        self._check(load().sph_read_state(self._h, field, C.c_void_p(out.data_ptr()), nbytes, 0))
        return self._after_read(out)

    def sph_read_state_host(self, field: int, out):
        """Host read into a (pinned) CPU tensor; returns after the copy has completed."""
        nbytes = out.numel() * out.element_size()
        self._check(load().sph_read_state(self._h, field, C.c_void_p(out.data_ptr()), nbytes, 1))
        return out

    def sph_read_state_host_async(self, field: int, out):
        """Asynchronous host read into a PINNED CPU tensor (is_host = 2): valid after sph_host_sync()."""
        assert out.is_pinned()
        nbytes = out.numel() * out.element_size()
        self._check(load().sph_read_state(self._h, field, C.c_void_p(out.data_ptr()), nbytes, 2))
        return out

    def sph_write_state_host_async(self, field: int, src):
        """Asynchronous host write from a PINNED CPU tensor (is_host = 2); the tensor must stay untouched until
        sph_host_sync() or the next step has consumed it."""
        assert src.is_pinned() and src.is_contiguous()
        nbytes = src.numel() * src.element_size()
        self._check(load().sph_write_state(self._h, field, C.c_void_p(src.data_ptr()), nbytes, 2))

    def sph_host_sync(self):
        self._check(load().sph_host_sync(self._h))

    def sph_write_state(self, field: int, src):
        t = self._torch
        if field == RIGID_BODIES:
            arr = make_bodies(src)
            self._check(load().sph_write_state(self._h, field, arr, C.sizeof(SphRigidBody) * self.nbodies, 1))
            return
        is_host = 0 if src.is_cuda else 1
        src = src.contiguous()
        nbytes = src.numel() * src.element_size()
        if not is_host:
            self._stream.wait_stream(t.cuda.current_stream(self.device))
            src.record_stream(self._stream)
        self._check(load().sph_write_state(self._h, field, C.c_void_p(src.data_ptr()), nbytes, is_host))

    def read_bodies(self):
        arr = (SphRigidBody * max(1, self.nbodies))()
        if self.nbodies:
            self._check(load().sph_read_state(self._h, RIGID_BODIES, arr, C.sizeof(SphRigidBody) * self.nbodies, 1))
        out = []
        for i in range(self.nbodies):
            b = arr[i]
            out.append(dict(first_particle=b.first_particle, n_particles=b.n_particles, dynamic=b.dynamic,
                            mass=b.mass, inertia_body=tuple(b.inertia_body[:]), com=tuple(b.com[:]),
                            quat=tuple(b.quat[:]), lin_vel=tuple(b.lin_vel[:]), ang_vel=tuple(b.ang_vel[:]),
                            contact_radius=b.contact_radius))
        return out

    def sph_read_stats(self) -> Dict[str, float]:
        s = SphStats()
        self._check(load().sph_read_stats(self._h, C.byref(s)))
        return {k: getattr(s, k) for k, _ in SphStats._fields_}

    def sph_enable_kernel_timing(self, enable: bool = True):
        self._check(load().sph_enable_kernel_timing(self._h, int(enable)))

    def sph_read_kernel_times(self) -> Dict[str, tuple]:
        """{kernel name: (launches, total ms)} since the last call."""
        buf = C.create_string_buffer(1 << 16)
        self._check(load().sph_read_kernel_times(self._h, buf, len(buf)))
        out = {}
        for line in buf.value.decode().splitlines():
            name, n, ms = line.split()
            out[name] = (int(n), float(ms))
        return out

    def sph_surface_extract(self, grid_min, dims, cube_size: float, iso: float = 0.6, max_triangles: int = 0):
        """Colour field + marching cubes (include/sph.h).  Returns (phi [nz, ny, nx] CUDA tensor, triangles
        [n, 3, 3] CUDA tensor, n_total); with max_triangles = 0 a first call counts the triangles and a second one
        emits exactly that many."""
        t = self._torch
        sp = SphSurfaceParams()
        sp.grid_min = (C.c_float * 3)(*[float(v) for v in grid_min])
        sp.dims = (C.c_int * 3)(*[int(v) for v in dims])
        sp.cube_size = float(cube_size); sp.iso = float(iso)
        nbytes = int(load().sph_surface_workspace_bytes(C.byref(sp)))
        if nbytes == 0:
            raise SphError(SPH_EINVAL, "sph_surface_workspace_bytes rejected the grid")
        ws = t.empty(nbytes + 256, dtype=t.uint8, device=self.device)
        off = (-ws.data_ptr()) % 256
        wptr = ws.data_ptr() + off
        self._stream.wait_stream(t.cuda.current_stream(self.device))
        ws.record_stream(self._stream)
        n = C.c_longlong(0)
        if max_triangles <= 0:
            self._check(load().sph_surface_extract(self._h, C.byref(sp), C.c_void_p(wptr), nbytes, None, 0, C.byref(n)))
            max_triangles = int(n.value)
        tris = t.empty((max(max_triangles, 1), 3, 3), dtype=t.float32, device=self.device)
        tris.record_stream(self._stream)
        self._check(load().sph_surface_extract(self._h, C.byref(sp), C.c_void_p(wptr), nbytes,
                                               C.c_void_p(tris.data_ptr()), max_triangles, C.byref(n)))
        nn = int(dims[0]) * int(dims[1]) * int(dims[2])
        phi = ws[off:off + 4 * nn].view(t.float32).reshape(int(dims[2]), int(dims[1]), int(dims[0]))
        return self._after_read(phi), self._after_read(tris[:min(int(n.value), max_triangles)]), int(n.value)

    def sph_render_particles(self, origin, right, up, pixel_size: float, width: int, height: int, radius: float = 0.0,
                             light=(0.0, 0.0, 0.0)):
        """Orthographic sphere-splat image of the fluid particles (include/sph.h, reading R30).  Returns CUDA tensors
        depth [H, W] float32 (+inf: empty), id [H, W] int32 (-1: empty), shade [H, W] float32.  light: the direction the
        light travels; the zero vector (default) is a headlight along the view direction."""
        t = self._torch
        rp = SphRenderParams()
        rp.origin = (C.c_float * 3)(*[float(v) for v in origin])
        rp.right = (C.c_float * 3)(*[float(v) for v in right])
        rp.up = (C.c_float * 3)(*[float(v) for v in up])
        rp.pixel_size = float(pixel_size); rp.width = int(width); rp.height = int(height); rp.radius = float(radius)
        rp.light = (C.c_float * 3)(*[float(v) for v in light])
        nbytes = int(load().sph_render_workspace_bytes(C.byref(rp), self.nf))
        if nbytes == 0:
            raise SphError(SPH_EINVAL, "sph_render_workspace_bytes rejected the camera")
        ws = t.empty(nbytes + 256, dtype=t.uint8, device=self.device)
        wptr = ws.data_ptr() + (-ws.data_ptr()) % 256
        depth = t.empty((int(height), int(width)), dtype=t.float32, device=self.device)
        pid = t.empty((int(height), int(width)), dtype=t.int32, device=self.device)
        shade = t.empty((int(height), int(width)), dtype=t.float32, device=self.device)
        self._stream.wait_stream(t.cuda.current_stream(self.device))
        for x in (ws, depth, pid, shade):
            x.record_stream(self._stream)
        self._check(load().sph_render_particles(self._h, C.byref(rp), C.c_void_p(wptr), nbytes, C.c_void_p(depth.data_ptr()),
                                                C.c_void_p(pid.data_ptr()), C.c_void_p(shade.data_ptr())))
        return self._after_read(depth), self._after_read(pid), self._after_read(shade)

    # ---- slab mode (include/sph.h): raw device pointers in, argument marshalling only
    def sph_slab_set_particles(self, pos4, vel4, n_owned: int, n_ghost: int):
        self._check(load().sph_slab_set_particles(self._h, C.c_void_p(pos4.data_ptr()), C.c_void_p(vel4.data_ptr()),
                                                  int(n_owned), int(n_ghost)))
        self.nf = int(n_owned) + int(n_ghost)

    def sph_slab_phase(self, phase: int):
        self._check(load().sph_slab_phase(self._h, int(phase)))

    def sph_slab_gather(self, field: int, orig_idx, n: int, out4):
        self._check(load().sph_slab_gather(self._h, int(field), C.c_void_p(orig_idx.data_ptr()), int(n), C.c_void_p(out4.data_ptr())))

    def sph_slab_scatter(self, field: int, first_orig: int, n: int, in4):
        self._check(load().sph_slab_scatter(self._h, int(field), int(first_orig), int(n), C.c_void_p(in4.data_ptr())))

    def sph_slab_read_error_sum(self) -> int:
        v = C.c_ulonglong(0)
        self._check(load().sph_slab_read_error_sum(self._h, C.byref(v)))
        return int(v.value)

    def sph_slab_set_loop(self, mode: int, cont: int, it: int, err: float):
        self._check(load().sph_slab_set_loop(self._h, int(mode), int(cont), int(it), float(err)))

    def sph_slab_store(self):
        """(pos4 ptr, vel4 ptr, orig_idx ptr, n, n_owned): device pointers into the workspace."""
        a, b, c = C.c_void_p(), C.c_void_p(), C.c_void_p()
        n, no = C.c_int(0), C.c_int(0)
        self._check(load().sph_slab_store(self._h, C.byref(a), C.byref(b), C.byref(c), C.byref(n), C.byref(no)))
        return a.value, b.value, c.value, int(n.value), int(no.value)

    def sph_launch_count(self) -> int:
        return int(load().sph_launch_count(self._h))

    def sph_destroy(self):
        if getattr(self, "_h", None):
            load().sph_destroy(self._h)
            self._h = None
            self._ws = None

    close = sph_destroy

    def __del__(self):
        try:
            self.sph_destroy()
        except Exception:
            pass
