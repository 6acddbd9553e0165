"""rflbm_diagnostics_static: the diagnostics for callers that cannot allocate device memory (include/rflbm.h).

Some users of this library hold a population field on the GPU but have no way to get the tens of gigabytes of workspace
that a handle (and with it rflbm_diagnostics) needs: a monitor or restart tool inside a simulation that has taken all of
the HBM, a plug-in that may not touch its host application's memory pool, code on a path where cudaMalloc's device-wide
synchronisation is off limits.  Their entry point keeps its reduction scratch in a static 2.5 MiB __device__ array of the
library and allocates nothing; it serves at most 2**27 sites.  These tests check it against the existing path
(Rflbm.diagnostics on the handle the field came from) on calls in a row that share the static array, and check the
size limit.  The file is named so that pytest collects it last: `pytest -x` stops at the first failure, and a failure
here must not hide the parity tests.
"""
import ctypes as C

import numpy as np
import pytest

from paper_2507_08820_b200 import binding, build, synthetic


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load()


def test_static_limit_and_argument_errors_are_host_side(lib):
    """No GPU needed: a refused call returns before any CUDA work, with a message that names the limit."""
    assert lib.rflbm_static_max_sites() == 2 ** 27
    out, err = (C.c_double * 10)(), C.create_string_buffer(512)
    # one site too many in z: 512 x 512 x 513
    rc = lib.rflbm_diagnostics_static(0x1000, 512, 512, 513, binding.F64, 0, None, None, out, err, len(err))
    assert rc == binding.EINVAL
    assert b"134217728" in err.value and b"exceeds" in err.value
    # the message buffer is optional
    assert lib.rflbm_diagnostics_static(0x1000, 2048, 2048, 2048, binding.F64, 0, None, None, out, None, 0) == binding.EINVAL
    assert lib.rflbm_diagnostics_static(None, 4, 4, 4, binding.F64, 0, None, None, out, err, len(err)) == binding.EINVAL
    assert b"NULL" in err.value
    assert lib.rflbm_diagnostics_static(0x1000, 4, 4, 4, binding.F64, 0, None, None, None, err, len(err)) == binding.EINVAL
    assert lib.rflbm_diagnostics_static(0x1000, 0, 4, 4, binding.F64, 0, None, None, out, err, len(err)) == binding.EINVAL
    assert lib.rflbm_diagnostics_static(0x1000, 4, 4, 4, 7, 0, None, None, out, err, len(err)) == binding.EINVAL
    assert lib.rflbm_diagnostics_static(0x1000, 4, 4, 2, binding.F64, 1, None, None, out, err, len(err)) == binding.EINVAL
    bad_g = (C.c_double * 3)(0.0, float("nan"), 0.0)
    assert lib.rflbm_diagnostics_static(0x1000, 4, 4, 4, binding.F64, 0, bad_g, None, out, err, len(err)) == binding.EINVAL


def _state(shape, prec, walls=False, g=None, scheme=binding.SCHEME_AB, steps=3, seed=5):
    """a handle a few noisy steps away from a smooth start: (handle, its canonical populations)"""
    import torch
    nx, ny, nz = shape
    sim = binding.Rflbm(nx, ny, nz, 0.8, 1e-4, 1.0, seed, prec, scheme=scheme)
    if walls:
        sim.set_walls_z(True)
    if g is not None:
        sim.set_force(*g)
    rho, u = synthetic.smooth_random_fields(nx, ny, nz, seed)
    sim.init(torch.from_numpy(rho), torch.from_numpy(u))
    sim.step(steps)
    return sim, sim.get_populations()


def _close(a, b):
    # the tolerance tests/test_gpu_parity.py uses between two GPU reductions of the same state (summation order differs)
    return np.allclose(a, b, rtol=1e-12, atol=1e-12)


@pytest.mark.gpu
def test_static_diagnostics_match_the_handle_on_calls_in_a_row():
    import torch
    # call 1: ten 4096-site chunks with a ragged tail, fp64, periodic
    big, f_big = _state((130, 33, 9), binding.F64)
    # call 2: ONE chunk, so rows 1..9 of the static array still hold call 1's partial sums and must not be read;
    #         fp32 storage, walls, body force, in-place AA scheme after an odd number of steps
    g = (1e-6, -2e-6, 0.0)
    small, f_small = _state((33, 5, 6), binding.F32, walls=True, g=g, scheme=binding.SCHEME_AA, steps=3)
    d_big = np.array(big.diagnostics())
    d_small = np.array(small.diagnostics())
    # The first call on a device is the set-up call: the CUDA runtime loads the library's module lazily, which is when
    # the 2.5 MiB static array and the two kernels get their device memory, and the call looks up the array's address.
    # From then on the free memory of the device must not move.
    s0 = np.array(binding.diagnostics_static(f_small, walls=True, g=g))
    free_before = torch.cuda.mem_get_info()[0]
    s1 = np.array(binding.diagnostics_static(f_big))
    s2 = np.array(binding.diagnostics_static(f_small, walls=True, g=g))
    s3 = np.array(binding.diagnostics_static(f_big))
    s4 = np.array(binding.diagnostics_static(f_small, walls=True, g=g))
    assert torch.cuda.mem_get_info()[0] == free_before            # nothing was allocated (or freed) on the device by the four calls
    assert np.array_equal(s0, s2)
    assert _close(s1, d_big), (s1, d_big)
    assert _close(s2, d_small), (s2, d_small)
    # fixed summation order: a repeated call returns the same bits, whatever ran in between
    assert np.array_equal(s1, s3) and np.array_equal(s2, s4)
    # and the numbers mean something: mass of a unit-density lattice, velocity variance of the noisy state > 0
    assert abs(s1[0] / (130 * 33 * 9) - 1.0) < 1e-3 and s1[7] > 0
    assert abs(s2[0] / (33 * 5 * 4) - 1.0) < 1e-3


@pytest.mark.gpu
def test_static_diagnostics_on_another_stream_and_bad_pointers():
    import torch
    sim, f = _state((64, 64, 33), binding.F64, steps=2)          # 33 chunks: more rows than one warp pass of stage 2
    d = np.array(sim.diagnostics())
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    s = np.array(binding.diagnostics_static(f, stream=st))
    assert _close(s, d), (s, d)
    # host memory is refused, not dereferenced
    lib = binding.load()
    host = torch.zeros(27 * 64, dtype=torch.float64)
    out, err = (C.c_double * 10)(), C.create_string_buffer(512)
    rc = lib.rflbm_diagnostics_static(host.data_ptr(), 4, 4, 4, binding.F64, 0, None, None, out, err, len(err))
    assert rc == binding.EINVAL and err.value
    # the handle's own path is untouched by all this
    assert _close(np.array(sim.diagnostics()), d)
