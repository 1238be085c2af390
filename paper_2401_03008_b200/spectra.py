"""Isotropised one-dimensional spectra of a periodic 2-D field (Fig. 5: "spectral densities ... as a function
of k_perp = (k_x^2 + k_y^2)^(1/2) (1D isotropized spectra)").

Post-processing of a state the solver produced, not part of the time step: the transform is torch.fft (a library
FFT on whatever device the tensor lives on), the binning is a scatter-add.  Conventions: for a real field f on an
ny x nx periodic grid, F = fft2(f)/(nx ny), and the spectrum E(m) collects |F|^2 of all modes whose integer radius
round(|m|) equals m, m = 0 .. min(nx, ny)/2; sum_m E(m) (+ the modes beyond the largest full shell) = <f^2>
(Parseval).  m is the mode number of the unit box; in the paper's box of side 2 pi it is k_perp itself.
"""
import math


def isotropic_spectrum_2d(f):
    """E(m) of one 2-D field (torch tensor, shape (ny, nx) or (1, ny, nx)); float64 tensor of length min(nx,ny)//2+1."""
    import torch

    f = f.reshape(f.shape[-2], f.shape[-1]).to(torch.float64)
    ny, nx = f.shape
    F = torch.fft.fft2(f) / (nx * ny)
    p = (F.real * F.real + F.imag * F.imag).reshape(-1)
    mx = torch.fft.fftfreq(nx, d=1.0 / nx, device=f.device, dtype=torch.float64)
    my = torch.fft.fftfreq(ny, d=1.0 / ny, device=f.device, dtype=torch.float64)
    r = torch.sqrt(my[:, None] ** 2 + mx[None, :] ** 2)
    shell = torch.round(r).to(torch.int64).reshape(-1)
    nshell = min(nx, ny) // 2 + 1
    keep = shell < nshell
    out = torch.zeros(nshell, dtype=torch.float64, device=f.device)
    out.index_add_(0, shell[keep], p[keep])
    return out


def spectrum_of_vector(fx, fy):
    """E(m) of a vector field in the plane: the sum of the spectra of its two components."""
    return isotropic_spectrum_2d(fx) + isotropic_spectrum_2d(fy)


def fit_slope(E, m_lo, m_hi):
    """Least-squares slope of log E against log m over the shells m_lo <= m <= m_hi (a plain Python float)."""
    import torch

    m = torch.arange(m_lo, m_hi + 1, dtype=torch.float64)
    y = torch.log(E[m_lo:m_hi + 1].detach().to("cpu", torch.float64))
    x = torch.log(m)
    xm, ym = x.mean(), y.mean()
    return float(((x - xm) * (y - ym)).sum() / ((x - xm) ** 2).sum())


def log_bins(E, per_octave=4):
    """(m_centre, mean E) over logarithmic bins of the shells 1..len(E)-1: a short table for text output."""
    E = E.detach().to("cpu")
    n = E.numel() - 1
    edges, e = [], 1.0
    while e < n:
        edges.append(e)
        e *= 2.0 ** (1.0 / per_octave)
    edges.append(float(n) + 0.5)
    rows = []
    for lo, hi in zip(edges[:-1], edges[1:]):
        a, b = int(math.ceil(lo)), int(math.ceil(hi)) - 1
        if b >= a:
            rows.append((math.sqrt(a * max(b, a)), float(E[a:b + 1].mean())))
    return rows
