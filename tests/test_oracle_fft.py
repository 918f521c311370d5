"""Pins for the oracle's own FFT (oracle/dm_oracle.c: fft1d, fft2_inplace).

Nothing here calls the oracle to check the oracle: the expected values are the DFT
definition written out (reading A6: forward unnormalised exp(-2 pi i (u x + v y)/N),
inverse with 1/N^2, DC at [0,0]), closed forms, and numpy.fft as a library cross-check.
"""
import numpy as np
import pytest

import oracle


def brute_dft2(x, sign=-1.0):
    """O(N^4) 2-D DFT straight from the definition; rows = y (axis 0), cols = x (axis 1)."""
    n = x.shape[0]
    out = np.zeros_like(x, dtype=np.complex128)
    for v in range(n):
        for u in range(n):
            acc = 0.0 + 0.0j
            for y in range(n):
                for xx in range(n):
                    acc += x[y, xx] * np.exp(sign * 2j * np.pi * (v * y + u * xx) / n)
            out[v, u] = acc
    return out


@pytest.mark.parametrize("n", [8, 16])
def test_fft2_matches_bruteforce_definition(n, rng):
    x = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    assert np.abs(oracle.fft2(x) - brute_dft2(x)).max() < 1e-12
    assert np.abs(oracle.fft2(x, inverse=True) - brute_dft2(x, +1.0) / n ** 2).max() < 1e-13


def test_fft2_axis_convention_single_delta():
    # delta at (y=1, x=2): X[v,u] = exp(-2 pi i (v*1 + u*2)/N); a transposed or sign-flipped
    # transform fails this.
    n = 16
    x = np.zeros((n, n), complex)
    x[1, 2] = 1.0
    v, u = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
    want = np.exp(-2j * np.pi * (v * 1 + u * 2) / n)
    assert np.abs(oracle.fft2(x) - want).max() < 1e-13


@pytest.mark.parametrize("n", [8, 64, 256])
def test_fft2_delta_constant_parseval_roundtrip(n, rng):
    d = np.zeros((n, n), complex)
    d[0, 0] = 1.0
    assert np.abs(oracle.fft2(d) - 1.0).max() < 1e-13            # delta -> constant
    c = np.full((n, n), 2.5 - 1j)
    fc = oracle.fft2(c)
    assert abs(fc[0, 0] - (2.5 - 1j) * n * n) < 1e-9 * n * n       # constant -> delta
    fc[0, 0] = 0
    assert np.abs(fc).max() < 1e-9
    x = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    X = oracle.fft2(x)
    assert abs((np.abs(x) ** 2).sum() - (np.abs(X) ** 2).sum() / n ** 2) < 1e-10 * (np.abs(x) ** 2).sum()
    assert np.abs(oracle.fft2(X, inverse=True) - x).max() < 1e-13 * n


@pytest.mark.parametrize("n", [64, 128, 256, 512])
def test_fft2_against_numpy_library(n, rng):
    x = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    ref = np.fft.fft2(x)
    assert np.linalg.norm(oracle.fft2(x) - ref) / np.linalg.norm(ref) < 1e-14
    ref = np.fft.ifft2(x)
    assert np.linalg.norm(oracle.fft2(x, inverse=True) - ref) / np.linalg.norm(ref) < 1e-14


def test_fft2_linearity_and_shift_theorem(rng):
    n = 32
    x = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    y = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    a = 0.3 - 2j
    assert np.abs(oracle.fft2(a * x + y) - (a * oracle.fft2(x) + oracle.fft2(y))).max() < 1e-11
    # circular shift by (3 rows, 5 cols) multiplies the spectrum by a linear phase
    v, u = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
    want = oracle.fft2(x) * np.exp(-2j * np.pi * (3 * v + 5 * u) / n)
    assert np.abs(oracle.fft2(np.roll(x, (3, 5), axis=(0, 1))) - want).max() < 1e-11


def test_fft2_rejects_non_power_of_two():
    with pytest.raises(ValueError):
        oracle.fft2(np.zeros((12, 12), complex))


def test_float_yardstick_build_is_float():
    assert oracle.lib("f32").oracle_real_bytes() == 4
    assert oracle.lib("f64").oracle_real_bytes() == 8
