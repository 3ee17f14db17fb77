"""ctypes wrapper of the fp64 CPU oracle (oracle/sphref.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this.  It never
imports the CUDA package's binding and shares no code with it; scenes come in as
plain numpy arrays and a parameter dictionary.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Dict, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sphref.c")
_LIB = os.path.join(_HERE, "libsphref.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (fp64, no contraction, OpenMP over particles)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class Params(C.Structure):
    _fields_ = [
        ("particle_radius", C.c_double), ("support_radius", C.c_double),
        ("rest_density", C.c_double), ("particle_mass", C.c_double), ("dt", C.c_double),
        ("gravity", C.c_double * 3),
        ("domain_min", C.c_double * 3), ("domain_max", C.c_double * 3),
        ("tank_min", C.c_double * 3), ("tank_max", C.c_double * 3),
        ("viscosity_mode", C.c_int), ("kinematic_viscosity", C.c_double),
        ("cg_rel_tol", C.c_double), ("cg_max_iter", C.c_int),
        ("eta_density", C.c_double), ("min_iter_density", C.c_int), ("max_iter_density", C.c_int),
        ("eta_divergence", C.c_double), ("min_iter_divergence", C.c_int), ("max_iter_divergence", C.c_int),
        ("enable_divergence_solve", C.c_int), ("force_iterations", C.c_int),
        ("wcsph_stiffness", C.c_double), ("wcsph_exponent", C.c_double),
        ("cfl_factor", C.c_double), ("dt_min", C.c_double),
        ("warm_start", C.c_int), ("warm_start_factor", C.c_double),
        ("pcisph_min_iter", C.c_int), ("pcisph_max_iter", C.c_int),
    ]


# parameters that scenes need not spell out
_DEFAULTS = dict(cfl_factor=0.0, dt_min=0.0, warm_start=0, warm_start_factor=0.5, pcisph_min_iter=3, pcisph_max_iter=100)


class Body(C.Structure):
    _fields_ = [
        ("first_particle", C.c_int), ("n_particles", C.c_int), ("dynamic", C.c_int),
        ("mass", C.c_double), ("inertia_body", C.c_double * 3),
        ("com", C.c_double * 3), ("quat", C.c_double * 4),
        ("lin_vel", C.c_double * 3), ("ang_vel", C.c_double * 3),
        ("contact_radius", C.c_double),
    ]


class Stats(C.Structure):
    _fields_ = [("it_v", C.c_int), ("it_d", C.c_int), ("cg_iters", C.c_int), ("oob_count", C.c_int),
                ("err_v", C.c_double), ("err_rho", C.c_double), ("cg_residual", C.c_double),
                ("v_max", C.c_double), ("dt_last", C.c_double), ("sim_time", C.c_double)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        ip = C.POINTER(C.c_int)
        L.sphref_create.restype = C.c_void_p
        L.sphref_create.argtypes = [C.POINTER(Params), C.c_int, C.c_void_p, C.c_void_p, C.c_int,
                                    C.c_void_p, C.c_void_p, C.c_int, C.POINTER(Body)]
        L.sphref_set_forced_dt.argtypes = [C.c_void_p, C.c_double]
        L.sphref_set_forced_dt.restype = None
        L.sphref_destroy.argtypes = [C.c_void_p]
        for name in ("sphref_build_grid", "sphref_compute_density_alpha", "sphref_step_wcsph"):
            getattr(L, name).argtypes = [C.c_void_p]
            getattr(L, name).restype = C.c_int
        L.sphref_step_dfsph.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int]
        L.sphref_divergence_solve.argtypes = [C.c_void_p, C.c_void_p, C.c_int]
        L.sphref_density_solve.argtypes = [C.c_void_p, C.c_void_p, C.c_int]
        L.sphref_pcisph_solve.argtypes = [C.c_void_p, C.c_void_p, C.c_int]
        L.sphref_step_pcisph.argtypes = [C.c_void_p, C.c_int]
        L.sphref_pcisph_k.argtypes = [C.c_void_p]
        L.sphref_pcisph_k.restype = C.c_double
        L.sphref_implicit_viscosity_solve.argtypes = [C.c_void_p, C.c_void_p, C.c_int]
        L.sphref_explicit_viscosity_accel.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.sphref_viscosity_operator.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.sphref_rigid_step.argtypes = [C.c_void_p]
        L.sphref_set_state.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.sphref_set_state_f64.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.sphref_set_boundary_state.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.sphref_set_bodies.argtypes = [C.c_void_p, C.POINTER(Body)]
        L.sphref_get_bodies.argtypes = [C.c_void_p, C.POINTER(Body)]
        L.sphref_set_params.argtypes = [C.c_void_p, C.POINTER(Params)]
        L.sphref_set_warm_state.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.sphref_set_warm_state.restype = None
        for name in ("sphref_pos", "sphref_vel", "sphref_density", "sphref_alpha", "sphref_kappa",
                     "sphref_kr", "sphref_ksum_v", "sphref_ksum_d", "sphref_psi", "sphref_boundary_pos", "sphref_boundary_vel",
                     "sphref_boundary_force"):
            getattr(L, name).argtypes = [C.c_void_p]
            getattr(L, name).restype = dp
        L.sphref_cg_history.argtypes = [C.c_void_p, ip]
        L.sphref_cg_history.restype = dp
        L.sphref_mass.argtypes = [C.c_void_p]
        L.sphref_mass.restype = C.c_double
        L.sphref_get_stats.argtypes = [C.c_void_p, C.POINTER(Stats)]
        L.sphref_grid_dims.argtypes = [C.c_void_p, C.c_int, ip]
        for name in ("sphref_cell_start", "sphref_cell_of_particle", "sphref_neighbor_start",
                     "sphref_neighbor_idx"):
            getattr(L, name).argtypes = [C.c_void_p, C.c_int]
            getattr(L, name).restype = ip
        L.sphref_W.argtypes = [C.c_double, C.c_double]
        L.sphref_W.restype = C.c_double
        L.sphref_gradW.argtypes = [dp, C.c_double, dp]
        L.sphref_num_threads.restype = C.c_int
        _lib = L
    return _lib


def W(r: float, h: float) -> float:
    return float(lib().sphref_W(float(r), float(h)))


def gradW(d: Sequence[float], h: float) -> np.ndarray:
    a = (C.c_double * 3)(*[float(v) for v in d])
    o = (C.c_double * 3)()
    lib().sphref_gradW(a, float(h), o)
    return np.array([o[0], o[1], o[2]])


def num_threads() -> int:
    return int(lib().sphref_num_threads())


def make_params(prm: Dict[str, object]) -> Params:
    p = Params()
    for name, ctype in Params._fields_:
        val = prm.get(name, _DEFAULTS[name]) if name in _DEFAULTS else prm[name]
        if hasattr(ctype, "_length_"):
            setattr(p, name, ctype(*[float(v) for v in val]))
        else:
            setattr(p, name, val)
    return p


def make_bodies(bodies) -> "C.Array":
    arr = (Body * max(1, len(bodies)))()
    for i, b in enumerate(bodies):
        arr[i].first_particle = b.first_particle
        arr[i].n_particles = b.n_particles
        arr[i].dynamic = b.dynamic
        arr[i].mass = b.mass
        arr[i].inertia_body = (C.c_double * 3)(*b.inertia_body)
        arr[i].com = (C.c_double * 3)(*b.com)
        arr[i].quat = (C.c_double * 4)(*b.quat)
        arr[i].lin_vel = (C.c_double * 3)(*b.lin_vel)
        arr[i].ang_vel = (C.c_double * 3)(*b.ang_vel)
        arr[i].contact_radius = b.contact_radius
    return arr


class Sim:
    """One oracle simulation.  All getters return numpy COPIES in original id order."""

    def __init__(self, fluid_pos, fluid_vel, boundary_pos, boundary_body, bodies, params):
        L = lib()
        self.nf = int(len(fluid_pos))
        self.nb = int(len(boundary_pos))
        self.nbodies = len(bodies)
        self.params = dict(params)
        fp = np.ascontiguousarray(fluid_pos, dtype=np.float32).reshape(-1, 3)
        fv = np.ascontiguousarray(fluid_vel, dtype=np.float32).reshape(-1, 3)
        bp = np.ascontiguousarray(boundary_pos, dtype=np.float32).reshape(-1, 3)
        bb = np.ascontiguousarray(boundary_body, dtype=np.int32)
        self._p = make_params(self.params)
        self._bodies = make_bodies(bodies)
        self._h = L.sphref_create(C.byref(self._p), self.nf, fp.ctypes.data, fv.ctypes.data, self.nb,
                                  bp.ctypes.data, bb.ctypes.data, self.nbodies, self._bodies)
        if not self._h:
            raise RuntimeError("sphref_create failed")

    @classmethod
    def from_scene(cls, scene, **overrides):
        prm = dict(scene.params)
        prm.update(overrides)
        return cls(scene.fluid_pos, scene.fluid_vel, scene.boundary_pos, scene.boundary_body,
                   scene.bodies, prm)

    def close(self):
        if getattr(self, "_h", None):
            lib().sphref_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- steps and pieces
    def update_params(self, **kw):
        self.params.update(kw)
        self._p = make_params(self.params)
        lib().sphref_set_params(self._h, C.byref(self._p))

    def build_grid(self):
        lib().sphref_build_grid(self._h)

    def compute_density_alpha(self):
        if lib().sphref_compute_density_alpha(self._h) != 0:
            raise RuntimeError("build_grid() first")

    def step_dfsph(self, forced_v: int = -1, forced_d: int = -1, forced_cg: int = -1):
        lib().sphref_step_dfsph(self._h, forced_v, forced_d, forced_cg)

    def step_wcsph(self):
        lib().sphref_step_wcsph(self._h)

    def set_forced_dt(self, dt: float = 0.0):
        """dt > 0: every following step uses exactly this time step (parity runs hand over the GPU's
        choice); 0: the CFL rule of reading R26 decides (fixed dt when cfl_factor = 0)."""
        lib().sphref_set_forced_dt(self._h, float(dt))

    def _solve(self, fn, vel, forced):
        v = np.ascontiguousarray(vel, dtype=np.float64).copy()
        it = fn(self._h, v.ctypes.data, forced)
        return v.reshape(-1, 3), int(it)

    def divergence_solve(self, vel, forced: int = -1):
        return self._solve(lib().sphref_divergence_solve, vel, forced)

    def density_solve(self, vel, forced: int = -1):
        return self._solve(lib().sphref_density_solve, vel, forced)

    def pcisph_solve(self, vel, forced: int = -1):
        """PCISPH pressure loop (reading R28) on the given velocities; accumulated pressure in kappa()."""
        return self._solve(lib().sphref_pcisph_solve, vel, forced)

    def step_pcisph(self, forced: int = -1):
        lib().sphref_step_pcisph(self._h, forced)

    def pcisph_k(self) -> float:
        """delta dt^2 of reading R28 (prototype-lattice constant)."""
        return float(lib().sphref_pcisph_k(self._h))

    def implicit_viscosity_solve(self, vel, forced: int = -1):
        return self._solve(lib().sphref_implicit_viscosity_solve, vel, forced)

    def viscosity_operator(self, u):
        u = np.ascontiguousarray(u, dtype=np.float64)
        out = np.zeros_like(u)
        lib().sphref_viscosity_operator(self._h, u.ctypes.data, out.ctypes.data)
        return out.reshape(-1, 3)

    def explicit_viscosity_accel(self, vel, rho=None):
        v = np.ascontiguousarray(vel, dtype=np.float64)
        r = np.ascontiguousarray(self.density() if rho is None else rho, dtype=np.float64)
        out = np.zeros_like(v)
        lib().sphref_explicit_viscosity_accel(self._h, v.ctypes.data, r.ctypes.data, out.ctypes.data)
        return out.reshape(-1, 3)

    def rigid_step(self):
        lib().sphref_rigid_step(self._h)

    # ---- state
    def set_state(self, pos, vel):
        p = np.ascontiguousarray(pos)
        v = np.ascontiguousarray(vel)
        if p.dtype == np.float32:
            lib().sphref_set_state(self._h, p.ctypes.data, np.ascontiguousarray(v, dtype=np.float32).ctypes.data)
        else:
            p = np.ascontiguousarray(p, dtype=np.float64)
            v = np.ascontiguousarray(v, dtype=np.float64)
            lib().sphref_set_state_f64(self._h, p.ctypes.data, v.ctypes.data)

    def set_boundary_state(self, bpos, bvel):
        p = np.ascontiguousarray(bpos, dtype=np.float32)
        v = np.ascontiguousarray(bvel, dtype=np.float32)
        lib().sphref_set_boundary_state(self._h, p.ctypes.data, v.ctypes.data)

    def set_bodies(self, bodies):
        self._bodies = make_bodies(bodies)
        lib().sphref_set_bodies(self._h, self._bodies)

    def bodies(self):
        arr = (Body * max(1, self.nbodies))()
        lib().sphref_get_bodies(self._h, arr)
        out = []
        for i in range(self.nbodies):
            b = arr[i]
            out.append(dict(first_particle=b.first_particle, n_particles=b.n_particles, dynamic=b.dynamic,
                            mass=b.mass, inertia_body=np.array(b.inertia_body[:]), com=np.array(b.com[:]),
                            quat=np.array(b.quat[:]), lin_vel=np.array(b.lin_vel[:]),
                            ang_vel=np.array(b.ang_vel[:]), contact_radius=b.contact_radius))
        return out

    def _arr(self, fn, n, cols=None):
        ptr = fn(self._h)
        a = np.ctypeslib.as_array(ptr, shape=(n * (cols or 1),)).copy()
        return a.reshape(n, cols) if cols else a

    def pos(self): return self._arr(lib().sphref_pos, self.nf, 3)
    def vel(self): return self._arr(lib().sphref_vel, self.nf, 3)
    def density(self): return self._arr(lib().sphref_density, self.nf)
    def alpha(self): return self._arr(lib().sphref_alpha, self.nf)
    def kappa(self): return self._arr(lib().sphref_kappa, self.nf)
    def ksum_v(self): return self._arr(lib().sphref_ksum_v, self.nf)
    def ksum_d(self): return self._arr(lib().sphref_ksum_d, self.nf)

    def set_warm_state(self, ksum_v, ksum_d):
        """Total stiffness of the last step's divergence / density solve (reading R27), id order."""
        a = np.ascontiguousarray(ksum_v, dtype=np.float64)
        b = np.ascontiguousarray(ksum_d, dtype=np.float64)
        assert a.shape == (self.nf,) and b.shape == (self.nf,)
        lib().sphref_set_warm_state(self._h, a.ctypes.data, b.ctypes.data)
    def psi(self): return self._arr(lib().sphref_psi, self.nb) if self.nb else np.zeros(0)
    def boundary_pos(self): return self._arr(lib().sphref_boundary_pos, self.nb, 3) if self.nb else np.zeros((0, 3))
    def boundary_vel(self): return self._arr(lib().sphref_boundary_vel, self.nb, 3) if self.nb else np.zeros((0, 3))
    def boundary_force(self): return self._arr(lib().sphref_boundary_force, self.nb, 3) if self.nb else np.zeros((0, 3))
    def mass(self): return float(lib().sphref_mass(self._h))

    def stats(self) -> Dict[str, float]:
        s = Stats()
        lib().sphref_get_stats(self._h, C.byref(s))
        return {k: getattr(s, k) for k, _ in Stats._fields_}

    def cg_history(self) -> np.ndarray:
        n = C.c_int(0)
        ptr = lib().sphref_cg_history(self._h, C.byref(n))
        return np.ctypeslib.as_array(ptr, shape=(n.value,)).copy()

    def grid_dims(self, which: int = 0):
        d = (C.c_int * 4)()
        lib().sphref_grid_dims(self._h, which, d)
        return tuple(d[:])

    def cell_start(self, which: int = 0) -> np.ndarray:
        nc = self.grid_dims(which)[3]
        return np.ctypeslib.as_array(lib().sphref_cell_start(self._h, which), shape=(nc + 1,)).copy()

    def cell_of_particle(self, which: int = 0) -> np.ndarray:
        n = self.nb if which else self.nf
        if n == 0:
            return np.zeros(0, dtype=np.int32)
        return np.ctypeslib.as_array(lib().sphref_cell_of_particle(self._h, which), shape=(n,)).copy()

    def neighbors(self, which: int = 0):
        """CSR (start[nf+1], idx) of fluid (0) or boundary (1) neighbours of every fluid particle,
        ids ascending within a row."""
        st = np.ctypeslib.as_array(lib().sphref_neighbor_start(self._h, which), shape=(self.nf + 1,)).copy()
        tot = int(st[-1])
        if tot == 0:
            return st, np.zeros(0, dtype=np.int32)
        idx = np.ctypeslib.as_array(lib().sphref_neighbor_idx(self._h, which), shape=(tot,)).copy()
        return st, idx
