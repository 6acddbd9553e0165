"""Seeded synthetic inputs shared by the tests, the smoke test and bench.py.

This module holds NONE of the method's arithmetic (no lattice tables, no equilibrium, no RNG of
the method): only initial density / velocity fields and raw random population vectors, as numpy
float64 arrays in the x-fastest layout rho[nz,ny,nx], u[3,nz,ny,nx].  Both the CUDA path and
the CPU oracle are fed from here so that they see identical inputs.
"""
from __future__ import annotations

import numpy as np


def uniform_fields(nx, ny, nz, rho0=1.0, u=(0.0, 0.0, 0.0)):
    """Uniform density and velocity (the paper's runs start from rho=1, u=0)."""
    rho = np.full((nz, ny, nx), float(rho0))
    uu = np.zeros((3, nz, ny, nx))
    for a in range(3):
        uu[a] = float(u[a])
    return rho, uu


def taylor_green_fields(nx, ny, nz, u0=0.01, rho0=1.0):
    """2-D Taylor-Green vortex, uniform in z (R15): wavevector 2*pi/nx in x and 2*pi/ny in y.
    u_x = u0 sin(kx x) cos(ky y), u_y = -u0 (kx/ky) cos(kx x) sin(ky y), rho = rho0."""
    kx = 2.0 * np.pi / nx
    ky = 2.0 * np.pi / ny
    x = np.arange(nx)[None, None, :]
    y = np.arange(ny)[None, :, None]
    rho = np.full((nz, ny, nx), float(rho0))
    u = np.zeros((3, nz, ny, nx))
    u[0] = u0 * np.sin(kx * x) * np.cos(ky * y)
    u[1] = -u0 * (kx / ky) * np.cos(kx * x) * np.sin(ky * y)
    return rho, u


def smooth_random_fields(nx, ny, nz, seed, rho0=1.0, drho=0.02, umax=0.03):
    """A few random low-order Fourier modes: non-trivial, smooth, low-Mach fields for parity tests."""
    rng = np.random.default_rng(seed)
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")

    def field():
        out = np.zeros((nz, ny, nx))
        for _ in range(4):
            m = rng.integers(-2, 3, size=3)
            ph = rng.uniform(0, 2 * np.pi)
            out += rng.uniform(-1, 1) * np.cos(2 * np.pi * (m[0] * x / nx + m[1] * y / ny + m[2] * z / nz) + ph)
        return out / 4.0

    rho = rho0 * (1.0 + drho * field())
    u = np.stack([umax * field() for _ in range(3)])
    return rho, u


def random_populations(seed, n=1, spread=0.05):
    """n random positive 27-vectors (arbitrary order, no lattice meaning): 1/27 * (1 + spread*U(-1,1))."""
    rng = np.random.default_rng(seed)
    return (1.0 + spread * rng.uniform(-1.0, 1.0, size=(n, 27))) / 27.0


def random_population_field(nx, ny, nz, seed, scale, spread=0.02):
    """Random population field f[27,nz,ny,nx] = scale[i] * (1 + spread*U(-1,1)); `scale` is supplied by the
    caller (e.g. lattice weights taken from whichever implementation is under test)."""
    rng = np.random.default_rng(seed)
    scale = np.asarray(scale, np.float64).reshape(27, 1, 1, 1)
    return scale * (1.0 + spread * rng.uniform(-1.0, 1.0, size=(27, nz, ny, nx)))


def gaussian_population_field(nx, ny, nz, seed, mean, std):
    """Independent Gaussian populations f[27,nz,ny,nx] = mean[i] + std[i] * N(0,1); `mean` and `std` (27 values each)
    are supplied by the caller (e.g. lattice weights and the thermal standard deviation of whichever implementation
    is under test): no lattice or physics constant lives here."""
    rng = np.random.default_rng(seed)
    mean = np.asarray(mean, np.float64).reshape(27, 1, 1, 1)
    std = np.asarray(std, np.float64).reshape(27, 1, 1, 1)
    return mean + std * rng.standard_normal(size=(27, nz, ny, nx))
