"""Host checks of the isotropised spectra used by the 2.5-D turbulence driver (Fig. 5): closed forms."""
import math

import numpy as np
import pytest
import torch

from paper_2401_03008_b200 import spectra


def grid(nx, ny):
    y, x = np.meshgrid((np.arange(ny) + 0.5) / ny, (np.arange(nx) + 0.5) / nx, indexing="ij")
    return x, y


def test_single_mode_lands_in_its_shell_with_half_its_amplitude_squared():
    nx, ny = 64, 48
    x, y = grid(nx, ny)
    f = 3.0 * np.cos(2 * np.pi * (3 * x - 4 * y) + 0.7)                  # |m| = 5
    E = spectra.isotropic_spectrum_2d(torch.from_numpy(f))
    assert E.numel() == 25
    assert float(E[5]) == pytest.approx(4.5, rel=1e-12)                 # A^2/2
    assert float(E.sum() - E[5]) <= 1e-24


def test_parseval_and_mean_in_shell_zero():
    rng = np.random.default_rng(1)
    f = rng.standard_normal((32, 32)) + 2.0
    E = spectra.isotropic_spectrum_2d(torch.from_numpy(f))
    F = np.fft.fft2(f) / f.size
    mx, my = np.meshgrid(np.fft.fftfreq(32, 1 / 32), np.fft.fftfreq(32, 1 / 32))
    inside = np.round(np.hypot(mx, my)) <= 16
    assert float(E.sum()) == pytest.approx(float((np.abs(F) ** 2)[inside].sum()), rel=1e-12)
    assert float(E[0]) == pytest.approx(f.mean() ** 2, rel=1e-12)
    assert float(E.sum()) <= (f ** 2).mean() + 1e-12                    # the corners of the square lie outside


def test_vector_spectrum_and_power_law_fit():
    n = 128
    x, y = grid(n, n)
    fx, fy = np.zeros((n, n)), np.zeros((n, n))
    for m in range(1, 41):                                              # one mode per shell, amplitude m^(-5/6)
        fx += m ** (-5.0 / 6.0) * np.cos(2 * np.pi * m * y + m)
        fy += 0.0
    E = spectra.spectrum_of_vector(torch.from_numpy(fx), torch.from_numpy(fy))
    for m in (1, 7, 40):
        assert float(E[m]) == pytest.approx(0.5 * m ** (-5.0 / 3.0), rel=1e-10)
    assert spectra.fit_slope(E, 2, 40) == pytest.approx(-5.0 / 3.0, abs=1e-10)
    rows = spectra.log_bins(E)
    assert rows[0][0] == 1.0 and rows[0][1] == pytest.approx(0.5, rel=1e-10)
    assert all(b[0] > a[0] for a, b in zip(rows, rows[1:]))
