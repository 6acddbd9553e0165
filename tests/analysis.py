"""Test-side numpy analysis shared by the oracle pins and the GPU physics tests (no oracle or CUDA code):
Taylor-Green amplitude, mode variances, spherically averaged structure factors (R11)."""
from __future__ import annotations

import numpy as np


def tg_amplitude(u, nx, ny):
    """A(t) = 4 <u_x sin(kx x) cos(ky y)> for the R15 vortex."""
    x = np.arange(nx)[None, None, :]
    y = np.arange(ny)[None, :, None]
    return 4.0 * np.mean(u[0] * np.sin(2 * np.pi * x / nx) * np.cos(2 * np.pi * y / ny))


def fit_decay_rate(t, a):
    """slope of -ln A vs t (least squares)."""
    t = np.asarray(t, float)
    la = np.log(np.asarray(a, float))
    return -np.polyfit(t, la, 1)[0]


def shell_spectrum(field, mean_sub=True):
    """|FFT|^2 / N binned by round(|k| L / 2 pi) (cubic box assumed for the shell index)."""
    f = field - field.mean() if mean_sub else field
    n = f.size
    p = np.abs(np.fft.fftn(f)) ** 2 / n
    idx = np.meshgrid(*[np.fft.fftfreq(s, 1.0 / s) for s in f.shape], indexing="ij")
    kk = np.sqrt(sum(i ** 2 for i in idx))
    shell = np.rint(kk).astype(int)
    nsh = shell.max() + 1
    tot = np.bincount(shell.ravel(), weights=p.ravel(), minlength=nsh)
    cnt = np.bincount(shell.ravel(), minlength=nsh)
    return tot, cnt


def shell_spectrum_torch(field, mean_sub=True):
    """shell_spectrum on the GPU (torch.fft): |FFT|^2 / N binned by round(|k| L / 2 pi); returns numpy (tot, cnt)."""
    import torch
    f = field.double()
    if mean_sub:
        f = f - f.mean()
    p = (torch.fft.fftn(f).abs() ** 2 / f.numel()).reshape(-1)
    axes = [torch.fft.fftfreq(s, 1.0 / s, device=f.device, dtype=torch.float64) for s in f.shape]
    kk = torch.sqrt(sum(a ** 2 for a in torch.meshgrid(*axes, indexing="ij")))
    shell = torch.round(kk).long().reshape(-1)
    nsh = int(shell.max()) + 1
    tot = torch.bincount(shell, weights=p, minlength=nsh)
    cnt = torch.bincount(shell, minlength=nsh)
    return tot.cpu().numpy(), cnt.cpu().numpy()
