"""Thin ctypes binding of the C-ABI library (include/rflbm.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of csrc/; PyTorch is used for device memory and
streams (the library itself never allocates device memory).  There is NO CPU fallback: if
csrc/librflbm.so is missing or CUDA is unavailable, construction raises.
"""
from __future__ import annotations

import ctypes as C
import os

F64, F32 = 0, 1
OK, EINVAL, ESTATE, ENOMEM, ECUDA = 0, -1, -2, -3, -4
KERNEL_AUTO, KERNEL_PLAIN, KERNEL_TMA = 0, 1, 2
MODEL_REG, MODEL_BGK = 0, 1
SCHEME_AB, SCHEME_AA = 0, 1
SIDE_LOW, SIDE_HIGH = 0, 1
Q = 27

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "csrc", "librflbm.so")
_lib = None

# every symbol include/rflbm.h declares: name -> (restype, argtypes)
_vp, _u64, _i32, _dbl, _sz = C.c_void_p, C.c_uint64, C.c_int, C.c_double, C.c_size_t
SYMBOLS = {
    "rflbm_create": (_i32, [_i32, _i32, _i32, _dbl, _dbl, _dbl, _u64, _i32, C.POINTER(_vp)]),
    "rflbm_workspace_bytes": (_sz, [_vp]),
    "rflbm_set_workspace": (_i32, [_vp, _vp, _sz]),
    "rflbm_set_stream": (_i32, [_vp, _vp]),
    "rflbm_set_walls_z": (_i32, [_vp, _i32]),
    "rflbm_set_force": (_i32, [_vp, _dbl, _dbl, _dbl]),
    "rflbm_set_kernel_variant": (_i32, [_vp, _i32]),
    "rflbm_set_model": (_i32, [_vp, _i32]),
    "rflbm_set_ghost_tau": (_i32, [_vp, _dbl]),
    "rflbm_set_scheme": (_i32, [_vp, _i32]),
    "rflbm_set_slab": (_i32, [_vp, _i32, _i32]),
    "rflbm_halo_bytes": (_sz, [_vp]),
    "rflbm_halo_pending": (_i32, [_vp]),
    "rflbm_halo_pack": (_i32, [_vp, _i32, _vp]),
    "rflbm_halo_unpack": (_i32, [_vp, _i32, _vp]),
    "rflbm_init": (_i32, [_vp, _vp, _vp]),
    "rflbm_step": (_i32, [_vp, _i32]),
    "rflbm_moments": (_i32, [_vp, _vp, _vp]),
    "rflbm_stress": (_i32, [_vp, _vp]),
    "rflbm_snapshot": (_i32, [_vp, _vp, _vp, _vp]),
    "rflbm_diagnostics": (_i32, [_vp, C.POINTER(_dbl)]),
    "rflbm_get_populations": (_i32, [_vp, _vp]),
    "rflbm_set_populations": (_i32, [_vp, _vp, _u64]),
    "rflbm_debug_rng": (_i32, [_vp, _u64, _vp, _vp]),
    "rflbm_run_host": (_i32, [_vp, _vp, _vp, _i32, _vp, _vp, _vp, _sz]),
    "rflbm_set_copy_stream": (_i32, [_vp, _vp]),
    "rflbm_debug_inject_failure": (_i32, [_vp, _i32]),
    "rflbm_launch_count": (_u64, [_vp]),
    "rflbm_last_kernel": (C.c_char_p, [_vp]),
    "rflbm_step_count": (_u64, [_vp]),
    "rflbm_last_error": (C.c_char_p, [_vp]),
    "rflbm_destroy": (_i32, [_vp]),
    "rflbm_static_max_sites": (C.c_longlong, []),
    "rflbm_diagnostics_static": (_i32, [_vp, _i32, _i32, _i32, _i32, _i32, C.POINTER(_dbl), _vp, C.POINTER(_dbl),
                                        C.c_char_p, _sz]),
}


class RflbmError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"rflbm error {code}: {msg}")
        self.code = code


def load():
    """dlopen csrc/librflbm.so (built by paper_2507_08820_b200.build); fails loudly if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2507_08820_b200.build` "
                           "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    for name, (res, args) in SYMBOLS.items():
        fn = getattr(lib, name)
        fn.restype = res
        fn.argtypes = args
    _lib = lib
    return lib


def _ptr(t):
    return 0 if t is None else t.data_ptr()


def diagnostics_static(f, walls=False, g=None, stream=None):
    """rflbm_diagnostics_static: the ten numbers of Rflbm.diagnostics() for a canonical population tensor
    f[27, nz, ny, nx] (CUDA, float64 or float32, contiguous) WITHOUT a handle or a workspace.

    For code that may not allocate device memory (a checkpoint inspector or monitor inside a process whose HBM is
    already taken, a plug-in that must stay out of the host's pool): the reduction scratch is a 2.5 MiB static array
    inside librflbm.so, so neither this wrapper nor the library allocates anything on the device.  At most
    rflbm_static_max_sites() = 2**27 sites; larger fields raise RflbmError(EINVAL).  Calls share the one array per GPU:
    do not overlap them (include/rflbm.h)."""
    import torch
    lib = load()
    assert f.is_cuda and f.is_contiguous() and f.dim() == 4 and f.shape[0] == Q, "f[27, nz, ny, nx] on the GPU"
    assert f.dtype in (torch.float64, torch.float32)
    nz, ny, nx = (int(v) for v in f.shape[1:])
    out, err = (_dbl * 10)(), C.create_string_buffer(512)
    gv = None if g is None else (_dbl * 3)(*(float(v) for v in g))
    with torch.cuda.device(f.device):
        st = stream if stream is not None else torch.cuda.current_stream(f.device)
        rc = lib.rflbm_diagnostics_static(f.data_ptr(), nx, ny, nz, F64 if f.dtype == torch.float64 else F32, int(bool(walls)),
                                          gv, st.cuda_stream, out, err, len(err))
    if rc != OK:
        raise RflbmError(rc, err.value.decode())
    return list(out)


class Rflbm:
    """One simulation handle.  Tensors are torch CUDA tensors in the x-fastest layout
    rho[nz,ny,nx], u[3,nz,ny,nx], f[27,nz,ny,nx] (canonical velocity order), dtype float64 or float32.

    Stream / device contract: every method runs under `torch.cuda.device(self.device)` and
    `torch.cuda.stream(self.stream)` (the stream given at construction, default: the stream current at construction),
    so the tensors it converts or allocates and the kernels the library enqueues are ordered on that one stream.
    A caller that consumes the returned tensors on another stream must order against `self.stream` itself.

    slab=(z0, nz_global): this handle owns layers [z0, z0+nz) of a global lattice (include/rflbm.h, rflbm_set_slab);
    init / set_populations then take fields with nz+2 layers and the halo_* methods move the faces."""

    def __init__(self, nx, ny, nz, tau, kT, rho0=1.0, seed=0, precision=F64, device="cuda:0", stream=None,
                 scheme=SCHEME_AB, slab=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("CUDA is not available: the rflbm path has no CPU fallback")
        self.torch = torch
        self.lib = load()
        self.nx, self.ny, self.nz = nx, ny, nz
        self.shape = (nz, ny, nx)
        self.shape_in = (nz + 2, ny, nx) if slab is not None else self.shape
        self.n = nx * ny * nz
        self.precision = precision
        self.dtype = torch.float64 if precision == F64 else torch.float32
        self.device = torch.device(device)
        h = _vp()
        rc = self.lib.rflbm_create(nx, ny, nz, tau, kT, rho0, seed, precision, C.byref(h))
        if rc != OK:
            raise RflbmError(rc, "rflbm_create: invalid argument")
        self.h = h
        if scheme != SCHEME_AB:
            self._ck(self.lib.rflbm_set_scheme(self.h, int(scheme)))
        if slab is not None:
            self._ck(self.lib.rflbm_set_slab(self.h, int(slab[0]), int(slab[1])))
        nbytes = self.lib.rflbm_workspace_bytes(self.h)
        with torch.cuda.device(self.device):
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)   # owned here, borrowed by C
            self._ck(self.lib.rflbm_set_workspace(self.h, self.workspace.data_ptr(), nbytes))
            self._ck(self.lib.rflbm_set_stream(self.h, self.stream.cuda_stream))

    def _ck(self, rc):
        if rc != OK:
            raise RflbmError(rc, self.lib.rflbm_last_error(self.h).decode())

    def _ctx(self):
        """device + stream of the handle for the duration of a call (see the class docstring)"""
        import contextlib
        st = contextlib.ExitStack()
        st.enter_context(self.torch.cuda.device(self.device))
        st.enter_context(self.torch.cuda.stream(self.stream))
        return st

    def close(self):
        if getattr(self, "h", None):
            self.lib.rflbm_destroy(self.h)
            self.h = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_walls_z(self, on=True):
        self._ck(self.lib.rflbm_set_walls_z(self.h, int(on)))

    def set_ghost_tau(self, tau_g):
        self._ck(self.lib.rflbm_set_ghost_tau(self.h, float(tau_g)))

    def set_model(self, model):
        self._ck(self.lib.rflbm_set_model(self.h, int(model)))

    def set_kernel_variant(self, variant):
        self._ck(self.lib.rflbm_set_kernel_variant(self.h, int(variant)))

    def set_force(self, gx, gy, gz):
        self._ck(self.lib.rflbm_set_force(self.h, gx, gy, gz))

    def _field(self, t, lead=(), shape=None):
        t = t.to(device=self.device, dtype=self.dtype).contiguous()
        shape = self.shape if shape is None else shape
        assert tuple(t.shape) == tuple(lead) + tuple(shape), (t.shape, lead, shape)
        return t

    def init(self, rho=None, u=None):
        with self._ctx():
            if rho is None:
                self._ck(self.lib.rflbm_init(self.h, None, None))
            else:
                rho, u = self._field(rho, (), self.shape_in), self._field(u, (3,), self.shape_in)
                self._ck(self.lib.rflbm_init(self.h, rho.data_ptr(), u.data_ptr()))
                self._keep = (rho, u)     # alive until the stream has consumed them

    def step(self, n=1):
        with self._ctx():
            self._ck(self.lib.rflbm_step(self.h, int(n)))

    def moments(self, rho=None, u=None):
        t = self.torch
        with self._ctx():
            if rho is None:
                rho = t.empty(self.shape, dtype=self.dtype, device=self.device)
                u = t.empty((3,) + self.shape, dtype=self.dtype, device=self.device)
            self._ck(self.lib.rflbm_moments(self.h, rho.data_ptr(), u.data_ptr()))
        return rho, u

    def stress(self, pi=None):
        with self._ctx():
            if pi is None:
                pi = self.torch.empty((6,) + self.shape, dtype=self.dtype, device=self.device)
            self._ck(self.lib.rflbm_stress(self.h, pi.data_ptr()))
        return pi

    def snapshot(self, rho=None, u=None, pi=None):
        """rho, u, pi of the current state from one pass over the populations (= moments() + stress(), bit for bit)"""
        t = self.torch
        with self._ctx():
            if rho is None:
                rho = t.empty(self.shape, dtype=self.dtype, device=self.device)
                u = t.empty((3,) + self.shape, dtype=self.dtype, device=self.device)
                pi = t.empty((6,) + self.shape, dtype=self.dtype, device=self.device)
            self._ck(self.lib.rflbm_snapshot(self.h, rho.data_ptr(), u.data_ptr(), pi.data_ptr()))
        return rho, u, pi

    def diagnostics(self):
        out = (_dbl * 10)()
        with self._ctx():
            self._ck(self.lib.rflbm_diagnostics(self.h, out))
        return list(out)

    def get_populations(self, f=None):
        with self._ctx():
            if f is None:
                f = self.torch.empty((Q,) + self.shape, dtype=self.dtype, device=self.device)
            self._ck(self.lib.rflbm_get_populations(self.h, f.data_ptr()))
        return f

    def set_populations(self, f, step=0):
        with self._ctx():
            f = self._field(f, (Q,), self.shape_in)
            self._ck(self.lib.rflbm_set_populations(self.h, f.data_ptr(), int(step)))
            self._keep = (f,)

    def debug_rng(self, step):
        t = self.torch
        with self._ctx():
            words = t.empty((24,) + self.shape, dtype=t.int32, device=self.device)
            normals = t.empty((23,) + self.shape, dtype=self.dtype, device=self.device)
            self._ck(self.lib.rflbm_debug_rng(self.h, int(step), words.data_ptr(), normals.data_ptr()))
        return words, normals

    def debug_inject_failure(self, nth_call):
        self._ck(self.lib.rflbm_debug_inject_failure(self.h, int(nth_call)))

    def set_copy_stream(self, stream):
        """second torch stream for the copies of run_host (None: serial)"""
        self._copy_stream = stream
        self._ck(self.lib.rflbm_set_copy_stream(self.h, stream.cuda_stream if stream is not None else None))

    def run_host(self, rho_host, u_host, nsteps, rho_out_host, u_out_host, scratch=None):
        """End-to-end job on HOST tensors (pinned for speed): upload, init, step, moments, download, sync;
        pipelined (time-skewed along z) when a copy stream has been set (include/rflbm.h)."""
        t = self.torch
        es = 8 if self.precision == F64 else 4
        with self._ctx():
            if scratch is None:
                scratch = t.empty(4 * self.n * es, dtype=t.uint8, device=self.device)
            self._ck(self.lib.rflbm_run_host(self.h, _ptr(rho_host), _ptr(u_host), int(nsteps), rho_out_host.data_ptr(),
                                             u_out_host.data_ptr(), scratch.data_ptr(), scratch.numel()))
        return rho_out_host, u_out_host

    # ---- slab faces (argument marshalling only; the CALLER moves the buffers between handles)
    @property
    def halo_bytes(self):
        return int(self.lib.rflbm_halo_bytes(self.h))

    @property
    def halo_pending(self):
        return bool(self.lib.rflbm_halo_pending(self.h))

    def halo_pack(self, side, face=None):
        with self._ctx():
            if face is None:
                face = self.torch.empty((9, self.ny, self.nx), dtype=self.dtype, device=self.device)
            self._ck(self.lib.rflbm_halo_pack(self.h, int(side), face.data_ptr()))
        return face

    def halo_unpack(self, side, face):
        with self._ctx():
            assert face.dtype == self.dtype and face.numel() == 9 * self.nx * self.ny and face.is_contiguous()
            self._ck(self.lib.rflbm_halo_unpack(self.h, int(side), face.data_ptr()))
            self._keep_face = getattr(self, "_keep_face", {})
            self._keep_face[side] = face

    @property
    def last_kernel(self):
        return self.lib.rflbm_last_kernel(self.h).decode()

    @property
    def step_count(self):
        return int(self.lib.rflbm_step_count(self.h))

    @property
    def launch_count(self):
        return int(self.lib.rflbm_launch_count(self.h))
