"""Pins for oracle O1 (the DFT of Eq. 2, readings G2/G3): closed forms, invariants and an
independent library FFT.  A wrong sign, a missing 1/m, a transposed axis or a bad twiddle fails here."""
import numpy as np
import pytest


def _rand(m, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal((m, m)) + 1j * rng.standard_normal((m, m))


@pytest.mark.parametrize("m", [2, 4, 8, 16, 32])
def test_radix2_equals_naive_definition(oracle, m):
    f = _rand(m, m)
    for sign in (-1, +1):
        assert np.abs(oracle.fft2(f, sign) - oracle.dft2_naive(f, sign)).max() < 1e-12


@pytest.mark.parametrize("m", [3, 5, 8])
def test_naive_matches_written_out_sum(oracle, m):
    # Eq. (2) typed out as a 4-index sum (G2 sign, 1/m scale); m need not be a power of two for the naive path
    f = _rand(m, 10 + m)
    u = np.arange(m)
    E = np.exp(-2j * np.pi * np.outer(u, u) / m)
    ref = np.einsum("ur,vc,rc->uv", E, E, f) / m
    assert np.abs(oracle.dft2_naive(f, -1) - ref).max() < 1e-12
    assert np.abs(oracle.dft2_naive(f, +1) - np.einsum("ur,vc,rc->uv", E.conj(), E.conj(), f) / m).max() < 1e-12


@pytest.mark.parametrize("m", [8, 64, 128])
def test_against_library_fft(oracle, m):
    f = _rand(m, 100 + m)
    assert np.abs(oracle.fft2(f, -1) - np.fft.fft2(f, norm="ortho")).max() < 1e-11
    assert np.abs(oracle.fft2(f, +1) - np.fft.ifft2(f, norm="ortho")).max() < 1e-11


def test_delta_closed_form_and_axes(oracle):
    # delta at (r0,c0) -> (1/m) exp(-2 pi i (u r0 + v c0)/m); r0 != c0 catches a transposed axis
    m, r0, c0 = 16, 3, 5
    f = np.zeros((m, m), complex); f[r0, c0] = 1.0
    u = np.arange(m)
    ref = np.exp(-2j * np.pi * (u[:, None] * r0 + u[None, :] * c0) / m) / m
    assert np.abs(oracle.fft2(f) - ref).max() < 1e-14
    assert np.abs(oracle.dft2_naive(f) - ref).max() < 1e-14


def test_dc_at_index_zero_and_unitary_scale(oracle):
    m = 32
    F1 = oracle.fft2(np.ones((m, m), complex))
    assert abs(F1[0, 0] - m) < 1e-12                      # (1/m) * m^2
    F1[0, 0] = 0
    assert np.abs(F1).max() < 1e-12


@pytest.mark.parametrize("m", [16, 64])
def test_parseval_inverse_linearity_shift(oracle, m):
    f, g = _rand(m, 1), _rand(m, 2)
    Ff = oracle.fft2(f)
    assert abs(np.linalg.norm(Ff) - np.linalg.norm(f)) < 1e-11 * np.linalg.norm(f)
    assert np.abs(oracle.fft2(Ff, +1) - f).max() < 1e-12                       # F* F = I
    assert np.abs(oracle.fft2(2 * f - 3j * g) - (2 * Ff - 3j * oracle.fft2(g))).max() < 1e-11
    # cyclic shift theorem: f(r - s) <-> exp(-2 pi i u s/m) F(u)
    s = (3, 7)
    u = np.arange(m)
    ph = np.exp(-2j * np.pi * (u[:, None] * s[0] + u[None, :] * s[1]) / m)
    assert np.abs(oracle.fft2(np.roll(f, s, axis=(0, 1))) - ph * Ff).max() < 1e-11


def test_adjointness_of_F(oracle):
    m = 16
    f, g = _rand(m, 3), _rand(m, 4)
    assert abs(np.vdot(oracle.fft2(f, -1), g) - np.vdot(f, oracle.fft2(g, +1))) < 1e-11
