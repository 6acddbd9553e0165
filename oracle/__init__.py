"""ctypes front end of the CPU oracle (oracle/rflbm_ref.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It imports nothing from
paper_2507_08820_b200 and shares no code with the CUDA path.

build() compiles the C file with gcc (-O2 -ffp-contract=off -fopenmp); load() returns the
ctypes library; Ref wraps one oracle handle with numpy host arrays (fp64 always).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "rflbm_ref.c")
_LIB = os.path.join(_HERE, "librflbm_ref.so")
_lib = None

Q = 27
F64, F32 = 0, 1
MODEL_REG, MODEL_BGK = 0, 1


def build(force: bool = False) -> str:
    """Compile the oracle if the shared object is missing or older than the source."""
    if (not force and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    cmd = ["gcc", "-std=c99", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared",
           "-o", _LIB, _SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return _LIB


def load():
    global _lib
    if _lib is not None:
        return _lib
    build()
    lib = C.CDLL(_LIB)
    vp, u64, i32, dbl = C.c_void_p, C.c_uint64, C.c_int, C.c_double
    pd = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
    pu32 = np.ctypeslib.ndpointer(dtype=np.uint32, flags="C_CONTIGUOUS")
    pi32 = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")
    lib.rflbm_ref_create.argtypes = [i32, i32, i32, dbl, dbl, dbl, u64, i32, C.POINTER(vp)]
    lib.rflbm_ref_create.restype = i32
    lib.rflbm_ref_destroy.argtypes = [vp]
    lib.rflbm_ref_set_threads.argtypes = [vp, i32]
    lib.rflbm_ref_max_threads.restype = i32
    lib.rflbm_ref_set_walls_z.argtypes = [vp, i32]
    lib.rflbm_ref_set_force.argtypes = [vp, dbl, dbl, dbl]
    lib.rflbm_ref_step_count.argtypes = [vp]
    lib.rflbm_ref_step_count.restype = u64
    lib.rflbm_ref_init.argtypes = [vp, vp, vp]
    lib.rflbm_ref_step.argtypes = [vp, i32]
    lib.rflbm_ref_step_reversed.argtypes = [vp, i32]
    lib.rflbm_ref_moments.argtypes = [vp, pd, pd]
    lib.rflbm_ref_diagnostics.argtypes = [vp, pd]
    lib.rflbm_ref_stress.argtypes = [vp, pd]
    lib.rflbm_ref_get_populations.argtypes = [vp, pd]
    lib.rflbm_ref_set_populations.argtypes = [vp, pd, u64]
    lib.rflbm_ref_debug_rng.argtypes = [vp, u64, pu32, pd]
    lib.rflbm_ref_tables.argtypes = [pi32, pd, pi32, pi32, pd, pd]
    lib.rflbm_ref_philox4x32_10.argtypes = [pu32, pu32, pu32]
    lib.rflbm_ref_philox4x32_10.restype = None
    lib.rflbm_ref_normal_pair.argtypes = [C.c_uint32, C.c_uint32, i32, pd]
    lib.rflbm_ref_normal_pair.restype = None
    lib.rflbm_ref_equilibrium.argtypes = [dbl, pd, pd]
    lib.rflbm_ref_equilibrium.restype = None
    lib.rflbm_ref_collide_site.argtypes = [pd, dbl, dbl, u64, i32, pd, C.c_uint32, u64, pd]
    lib.rflbm_ref_collide_site_bgk.argtypes = [pd, dbl, dbl, u64, i32, C.c_uint32, u64, pd]
    lib.rflbm_ref_set_model.argtypes = [vp, i32]
    lib.rflbm_ref_set_ghost_tau.argtypes = [vp, dbl]
    lib.rflbm_ref_collide_site_ghost.argtypes = [pd, dbl, dbl, dbl, u64, i32, C.c_uint32, u64, pd]
    lib.rflbm_ref_moments_of.argtypes = [pd, pd]
    lib.rflbm_ref_moments_of.restype = None
    _lib = lib
    return lib


def max_threads() -> int:
    return int(load().rflbm_ref_max_threads())


def tables():
    """(c[27,3], w[27], opp[27], pqr[27,3], e[27,27], b[27]) exactly as the oracle uses them."""
    lib = load()
    c = np.zeros((Q, 3), np.int32)
    w = np.zeros(Q)
    opp = np.zeros(Q, np.int32)
    pqr = np.zeros((Q, 3), np.int32)
    e = np.zeros((Q, Q))
    b = np.zeros(Q)
    lib.rflbm_ref_tables(c, w, opp, pqr, e, b)
    return c, w, opp, pqr, e, b


def philox(ctr, key):
    out = np.zeros(4, np.uint32)
    load().rflbm_ref_philox4x32_10(np.asarray(ctr, np.uint32), np.asarray(key, np.uint32), out)
    return out


def normal_pair(xa: int, xb: int, precision: int = F64):
    out = np.zeros(2)
    load().rflbm_ref_normal_pair(int(xa), int(xb), precision, out)
    return out


def equilibrium(rho: float, u):
    out = np.zeros(Q)
    load().rflbm_ref_equilibrium(float(rho), np.ascontiguousarray(u, np.float64), out)
    return out


def collide_site(g, tau, kT=0.0, seed=0, precision=F64, gacc=(0.0, 0.0, 0.0), site=0, t=0):
    out = np.zeros(Q)
    load().rflbm_ref_collide_site(np.ascontiguousarray(g, np.float64), float(tau), float(kT), int(seed),
                                  precision, np.ascontiguousarray(gacc, np.float64), int(site), int(t), out)
    return out


def collide_site_ghost(g, tau, tau_g, kT=0.0, seed=0, precision=F64, site=0, t=0):
    """Reg-FLBM collision with a general ghost relaxation time (Eq.21 live)."""
    out = np.zeros(Q)
    load().rflbm_ref_collide_site_ghost(np.ascontiguousarray(g, np.float64), float(tau), float(tau_g), float(kT),
                                        int(seed), precision, int(site), int(t), out)
    return out


def collide_site_bgk(g, tau, kT=0.0, seed=0, precision=F64, site=0, t=0):
    """BGK-FLBM (Eq.11) collision of one site."""
    out = np.zeros(Q)
    load().rflbm_ref_collide_site_bgk(np.ascontiguousarray(g, np.float64), float(tau), float(kT), int(seed),
                                      precision, int(site), int(t), out)
    return out


def moments_of(f):
    out = np.zeros(Q)
    load().rflbm_ref_moments_of(np.ascontiguousarray(f, np.float64), out)
    return out


class RefError(RuntimeError):
    pass


class Ref:
    """One oracle simulation.  Arrays are numpy float64, x fastest: rho[nz,ny,nx], u[3,nz,ny,nx],
    f[27,nz,ny,nx] in the canonical velocity order (R1)."""

    def __init__(self, nx, ny, nz, tau, kT, rho0=1.0, seed=0, precision=F64, threads=1):
        self.lib = load()
        self.shape = (nz, ny, nx)
        self.n = nx * ny * nz
        h = C.c_void_p()
        rc = self.lib.rflbm_ref_create(nx, ny, nz, tau, kT, rho0, seed, precision, C.byref(h))
        if rc != 0:
            raise RefError(f"rflbm_ref_create -> {rc}")
        self.h = h
        self.lib.rflbm_ref_set_threads(self.h, max(1, int(threads)))

    def _ck(self, rc, what):
        if rc != 0:
            raise RefError(f"{what} -> {rc}")

    def close(self):
        if getattr(self, "h", None):
            self.lib.rflbm_ref_destroy(self.h)
            self.h = None

    def __del__(self):
        self.close()

    def set_walls_z(self, on=True):
        self._ck(self.lib.rflbm_ref_set_walls_z(self.h, int(on)), "set_walls_z")

    def set_ghost_tau(self, tau_g):
        self._ck(self.lib.rflbm_ref_set_ghost_tau(self.h, float(tau_g)), "set_ghost_tau")

    def set_model(self, model):
        self._ck(self.lib.rflbm_ref_set_model(self.h, int(model)), "set_model")

    def set_force(self, gx, gy, gz):
        self._ck(self.lib.rflbm_ref_set_force(self.h, gx, gy, gz), "set_force")

    def init(self, rho=None, u=None):
        if rho is None:
            self._ck(self.lib.rflbm_ref_init(self.h, None, None), "init")
        else:
            rho = np.ascontiguousarray(rho, np.float64).reshape(self.shape)
            u = np.ascontiguousarray(u, np.float64).reshape((3,) + self.shape)
            self._ck(self.lib.rflbm_ref_init(self.h, rho.ctypes.data, u.ctypes.data), "init")

    def step(self, n=1):
        self._ck(self.lib.rflbm_ref_step(self.h, int(n)), "step")

    def step_reversed(self, n=1):
        self._ck(self.lib.rflbm_ref_step_reversed(self.h, int(n)), "step_reversed")

    @property
    def step_count(self):
        return int(self.lib.rflbm_ref_step_count(self.h))

    def moments(self):
        rho = np.zeros(self.shape)
        u = np.zeros((3,) + self.shape)
        self._ck(self.lib.rflbm_ref_moments(self.h, rho, u), "moments")
        return rho, u

    def stress(self):
        pi = np.zeros((6,) + self.shape)
        self._ck(self.lib.rflbm_ref_stress(self.h, pi), "stress")
        return pi

    def diagnostics(self):
        out = np.zeros(10)
        self._ck(self.lib.rflbm_ref_diagnostics(self.h, out), "diagnostics")
        return out

    def get_populations(self):
        f = np.zeros((Q,) + self.shape)
        self._ck(self.lib.rflbm_ref_get_populations(self.h, f), "get_populations")
        return f

    def set_populations(self, f, step=0):
        f = np.ascontiguousarray(f, np.float64).reshape((Q,) + self.shape)
        self._ck(self.lib.rflbm_ref_set_populations(self.h, f, int(step)), "set_populations")

    def debug_rng(self, step):
        words = np.zeros((24,) + self.shape, np.uint32)
        normals = np.zeros((23,) + self.shape)
        self._ck(self.lib.rflbm_ref_debug_rng(self.h, int(step), words, normals), "debug_rng")
        return words, normals
