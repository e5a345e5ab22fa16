"""Pins for oracle O6, O7, O9 and the reconstruction sequence: fixed point, the beta = 1
Douglas-Rachford special case, equality of the literal and one-split forms, the negative control for the
printed sign (reading G1), metric invariances, and convergence on a well-posed noise-free scan (PAPER.md:248
"all residuals decrease rapidly")."""
import dataclasses

import numpy as np
import pytest

import synth


def _rc(shape, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


def _small_scan(seed=0, m=16, K=20, shape=(40, 44)):
    rng = np.random.default_rng(seed)
    pos = np.stack([rng.integers(0, shape[0] - m + 1, K), rng.integers(0, shape[1] - m + 1, K)], 1).astype(np.int32)
    w = _rc((m, m), seed + 1) * np.exp(-((np.arange(m) - m / 2) ** 2)[:, None] / 30 - ((np.arange(m) - m / 2) ** 2)[None] / 30)
    psi = 0.5 + _rc(shape, seed + 2) * 0.3
    return m, K, shape, pos, w, psi


def test_raar_fixed_point_P4(oracle):
    m, K, shape, pos, w, psi = _small_scan()
    z0 = oracle.split(psi, w, pos)
    a = np.abs(np.fft.fft2(z0, norm="ortho"))
    for beta in (0.6, 0.75, 1.0):
        z1 = oracle.raar(z0, w, pos, shape, a, 1e-9, beta)
        assert np.abs(z1 - z0).max() < 1e-12
    e = oracle.errors(z0, z0, w, pos, shape, a, 1e-9, float((a ** 2).sum()))
    assert np.all(e < 1e-12)                                                           # P6: all zero there


@pytest.mark.parametrize("beta", [0.6, 0.75, 0.9, 1.0])
def test_raar_typed_out_and_forms_agree(oracle, beta):
    m, K, shape, pos, w, psi = _small_scan(1)
    z = _rc((K, m, m), 9)
    a = np.abs(_rc((K, m, m), 10)) + 0.05
    zn, y = oracle.raar(z, w, pos, shape, a, 1e-9, beta, return_y=True)
    # y is P_a z by the library FFT
    Z = np.fft.fft2(z, norm="ortho")
    y_ref = np.fft.ifft2(Z / np.abs(Z) * a, norm="ortho")
    assert np.abs(y - y_ref).max() < 1e-11
    # Luke's RAAR: beta/2 (R_Q R_a + I) z + (1 - beta) P_a z with reflectors R = 2P - I  ([60])
    PQ = lambda f: oracle.PQ(f, w, pos, shape)
    Ra = 2 * y_ref - z
    luke = 0.5 * beta * ((2 * PQ(Ra) - Ra) + z) + (1 - beta) * y_ref
    assert np.abs(zn - luke).max() < 1e-11
    assert np.abs(oracle.raar_one_split(z, w, pos, shape, a, 1e-9, beta) - zn).max() < 1e-12
    if beta == 1.0:   # Douglas-Rachford / difference map: z + P_Q(2 P_a z - z) - P_a z
        assert np.abs(zn - (z + PQ(2 * y_ref - z) - y_ref)).max() < 1e-11
    # identity L z' = L P_a z  (step 6 after step 5 with w unchanged)
    cov = oracle.cover_counts(m, pos, shape) > 0
    assert np.abs(oracle.L(zn, w, pos, shape)[cov] - oracle.L(y, w, pos, shape)[cov]).max() < 1e-11


def test_printed_sign_is_not_what_the_oracle_does_G1(oracle):
    # a component with P_a z = z and P_Q z = 0 is multiplied by (1 - beta) under Luke's sign and by (1 - 3 beta)
    # under the sign printed at PAPER.md:176
    m, K, shape, pos, w, psi = _small_scan(2)
    z = _rc((K, m, m), 3)
    z = z - oracle.PQ(z, w, pos, shape)                     # P_Q z = 0
    a = np.abs(np.fft.fft2(z, norm="ortho"))                # P_a z = z
    beta = 0.75
    zn = oracle.raar(z, w, pos, shape, a, 1e-12, beta)
    assert np.abs(zn - (1 - beta) * z).max() < 1e-11
    assert np.abs(zn - (1 - 3 * beta) * z).max() > 0.1


def test_metric_definitions_and_invariances_P6(oracle):
    m, K, shape, pos, w, psi = _small_scan(4)
    z, zp = _rc((K, m, m), 5), _rc((K, m, m), 6)
    a = np.abs(_rc((K, m, m), 7)) + 0.05
    A2 = float((a ** 2).sum())
    e = oracle.errors(z, zp, w, pos, shape, a, 1e-9, A2)
    Z = np.fft.fft2(z, norm="ortho")
    assert abs(e[0] - np.linalg.norm(a - np.abs(Z)) / np.sqrt(A2)) < 1e-11           # Eq. 11 via Parseval
    assert abs(e[1] - np.linalg.norm(oracle.PQ(z, w, pos, shape) - z) / np.sqrt(A2)) < 1e-12
    assert abs(e[2] - np.linalg.norm(z - zp) / np.sqrt(A2)) < 1e-12
    e0 = oracle.errors(z, None, w, pos, shape, a, 1e-9, A2)                           # G7: z^(l-1) = 0
    assert abs(e0[2] - np.linalg.norm(z) / np.sqrt(A2)) < 1e-12
    ph = np.exp(1.1j)
    assert np.abs(oracle.errors(ph * z, ph * zp, w, pos, shape, a, 1e-9, A2) - e).max() < 1e-11
    s = 3.0    # I -> s^2 I (a -> s a), frames -> s z : all metrics unchanged
    assert np.abs(oracle.errors(s * z, s * zp, w, pos, shape, s * a, s * 1e-9, s * s * A2) - e).max() < 1e-11


def test_sequence_matches_stepwise_calls_and_G10_order(oracle):
    cfg = synth.reduced(synth.config(1), 4)
    pos, shape, I, w0, obj, wt = synth.make(cfg)
    orc = oracle.Oracle(cfg.m, pos, shape, I, w0, refine_every=2)
    z = oracle.split(np.ones(shape, complex), w0.astype(complex), pos)
    assert np.array_equal(orc.z, z)                                                    # step 4, G7/G8
    assert abs(orc.errors()[2] - np.linalg.norm(z) / np.sqrt(orc.A2)) < 1e-12
    w = w0.astype(complex)
    for it in (1, 2, 3):
        z = oracle.raar(z, w, pos, shape, orc.a, orc.thr, 0.75)                        # old w
        psi = oracle.L(z, w, pos, shape)                                               # old w
        if it % 2 == 0:
            w = oracle.probe_update(psi, z, w, pos)                                    # new frames, that psi
        orc.iterate(1, 0.75)
        assert np.array_equal(orc.z, z) and np.array_equal(orc.w, w) and np.array_equal(orc.psi, psi)


def test_converges_on_a_well_posed_noise_free_scan(oracle):
    # broad probe, dense overlap, exact illumination, noise-free: "all residuals decrease rapidly"
    cfg = dataclasses.replace(synth.reduced(synth.config(1), 5), photons=0.0, step=12, phase_coeff=0.05)
    pos, shape, I, w0, obj, wt = synth.make(cfg)
    orc = oracle.Oracle(cfg.m, pos, shape, I, w0)
    e0 = orc.iterate(1, 0.75).errors()
    e1 = orc.iterate(99, 0.75).errors()
    assert np.all(e1 < 1e-4 * e0)
    # object agrees with the truth up to a global phase where it is well lit (Eq. 14 idea)
    den = oracle.overlap_den(orc.w, pos, shape)
    lit = den > 0.05 * den.max()
    rec, tru = orc.object()[lit], obj.astype(complex)[lit]
    ph = np.vdot(rec, tru); ph /= abs(ph)
    assert np.linalg.norm(ph * rec - tru) / np.linalg.norm(tru) < 1e-3          # eps_0 < 5e-4 scale
