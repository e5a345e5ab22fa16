"""Pins for oracle O2-O5, O8, O10: the split / overlap operators (Eq. 5 at :127, Eq. 8-10 at
:145-159), the data projector (Eq. 7 at :141-143) and the integer geometry, against things the oracle did not
compute itself: a dense matrix built from Eq. (5), numpy fancy indexing, closed-form special cases, projector
identities."""
import numpy as np
import pytest


def _rc(shape, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


def _dense_Q(w, pos, shape):
    """Eq. (5): the (K m^2) x (n_r n_c) matrix whose block i is diag(w) T_i."""
    m = w.shape[0]; nr, nc = shape; K = len(pos)
    Q = np.zeros((K * m * m, nr * nc), complex)
    for i, (pr, pc) in enumerate(pos):
        for r in range(m):
            for c in range(m):
                Q[(i * m + r) * m + c, (pr + r) * nc + (pc + c)] = w[r, c]
    return Q


TINY_POS = np.array([[0, 0], [1, 2], [3, 1], [2, 3]], dtype=np.int32)   # n=6, m=3, K=4


def test_split_is_the_matrix_of_eq5(oracle):
    m, shape = 3, (6, 6)
    w, psi = _rc((m, m), 1), _rc(shape, 2)
    Q = _dense_Q(w, TINY_POS, shape)
    z = oracle.split(psi, w, TINY_POS)
    assert np.abs(z.ravel() - Q @ psi.ravel()).max() < 1e-14


def test_overlap_is_the_adjoint_matrix_and_PQ_is_the_dense_projector(oracle):
    m, shape = 3, (6, 6)
    w, f = _rc((m, m), 3), _rc((4, m, m), 4)
    Q = _dense_Q(w, TINY_POS, shape)
    num = oracle.overlap_num(f, w, TINY_POS, shape)
    assert np.abs(num.ravel() - Q.conj().T @ f.ravel()).max() < 1e-13
    den = oracle.overlap_den(w, TINY_POS, shape)
    assert np.abs(den.ravel() - np.real(np.diag(Q.conj().T @ Q))).max() < 1e-13
    # Q*Q is diagonal (Eq. 9 divides point-wise): off-diagonal must vanish
    G = Q.conj().T @ Q
    assert np.abs(G - np.diag(np.diag(G))).max() == 0.0
    # P_Q = Q (Q*Q)^-1 Q*, Eq. (8), as the orthogonal projector onto range(Q) from an SVD-based pinv
    P = Q @ np.linalg.pinv(Q)
    assert np.abs(oracle.PQ(f, w, TINY_POS, shape).ravel() - P @ f.ravel()).max() < 1e-12


def test_uncovered_pixels_are_zero_G5(oracle):
    m, shape = 3, (6, 6)
    w, f = _rc((m, m), 5), _rc((4, m, m), 6)
    psi = oracle.L(f, w, TINY_POS, shape)
    cnt = oracle.cover_counts(m, TINY_POS, shape)
    assert (cnt == 0).any()
    assert np.all(psi[cnt == 0] == 0) and np.all(np.isfinite(psi))


@pytest.mark.parametrize("seed", [0, 1])
def test_adjointness_and_projector_identities(oracle, seed):
    rng = np.random.default_rng(seed)
    m, K, shape = 8, 12, (20, 23)                        # rectangular object catches a row/col stride mix-up
    pos = np.stack([rng.integers(0, shape[0] - m + 1, K), rng.integers(0, shape[1] - m + 1, K)], 1).astype(np.int32)
    w, psi, z = _rc((m, m), 10 + seed), _rc(shape, 20 + seed), _rc((K, m, m), 30 + seed)
    # <Q psi, z> = <psi, Q* z>  (pins T against T^T and where the conjugate goes)
    assert abs(np.vdot(oracle.split(psi, w, pos), z) - np.vdot(psi, oracle.overlap_num(z, w, pos, shape))) < 1e-10
    # split against numpy fancy indexing
    r = np.arange(m)
    ref = w[None] * psi[pos[:, 0, None, None] + r[None, :, None], pos[:, 1, None, None] + r[None, None, :]]
    assert np.abs(oracle.split(psi, w, pos) - ref).max() < 1e-14
    # Q*Q 1 = den ; P_Q idempotent, self-adjoint, fixes range(Q)
    one = np.ones(shape, complex)
    assert np.abs(oracle.overlap_num(oracle.split(one, w, pos), w, pos, shape).real
                  - oracle.overlap_den(w, pos, shape)).max() < 1e-12
    Pz = oracle.PQ(z, w, pos, shape)
    assert np.abs(oracle.PQ(Pz, w, pos, shape) - Pz).max() < 1e-12
    z2 = _rc((K, m, m), 40 + seed)
    assert abs(np.vdot(Pz, z2) - np.vdot(z, oracle.PQ(z2, w, pos, shape))) < 1e-10
    cov = oracle.cover_counts(m, pos, shape) > 0
    Qpsi = oracle.split(psi, w, pos)
    assert np.abs(oracle.PQ(Qpsi, w, pos, shape) - Qpsi).max() < 1e-12
    assert np.abs(oracle.L(Qpsi, w, pos, shape)[cov] - psi[cov]).max() < 1e-12


def test_mosaic_and_mean_special_cases(oracle):
    m, shape = 4, (8, 8)
    pos = np.array([[0, 0], [0, 4], [4, 0], [4, 4]], np.int32)
    f = _rc((4, m, m), 7)
    w1 = np.ones((m, m), complex)
    mosaic = np.block([[f[0], f[1]], [f[2], f[3]]])
    assert np.abs(oracle.overlap_num(f, w1, pos, shape) - mosaic).max() == 0.0
    assert np.all(oracle.overlap_den(w1, pos, shape) == 1.0)
    same = np.zeros((5, 2), np.int32)
    g = _rc((5, m, m), 8)
    assert np.abs(oracle.L(g, w1, same, (4, 4)) - g.mean(0)).max() < 1e-14


def test_amplitudes(oracle):
    I = np.array([[4.0, 0.25], [-1.0, 9.0]], np.float32)
    a, A2, a_rms, thr = oracle.amplitudes(I)
    assert np.all(a == np.array([[2.0, 0.5], [0.0, 3.0]]))                    # G14 clamp
    assert A2 == 13.25 and abs(a_rms - np.sqrt(13.25 / 4)) < 1e-15 and abs(thr - 1e-4 * a_rms) < 1e-18


def test_Pa_properties(oracle):
    rng = np.random.default_rng(3)
    K, m = 3, 16
    z = _rc((K, m, m), 11)
    a = rng.random((K, m, m)) + 0.1
    thr = 1e-6
    y = oracle.Pa(z, a, thr)
    # |F P_a z| = a, phase of F P_a z = phase of F z  (checked with the library FFT, not the oracle's)
    Y, Z = np.fft.fft2(y, norm="ortho"), np.fft.fft2(z, norm="ortho")
    assert np.abs(np.abs(Y) - a).max() < 1e-12
    assert np.abs(Y / np.abs(Y) - Z / np.abs(Z)).max() < 1e-10
    assert np.abs(oracle.Pa(y, a, thr) - y).max() < 1e-12                    # idempotent
    phi = np.exp(0.7j)
    assert np.abs(oracle.Pa(phi * z, a, thr) - phi * y).max() < 1e-12        # phase covariance
    assert abs(np.linalg.norm(y - z) - np.linalg.norm(a - np.abs(Z))) < 1e-10  # Parseval form of eps_a
    assert np.abs(oracle.Pa(z, np.abs(Z), thr) - z).max() < 1e-12            # a := |Fz| -> identity
    assert np.abs(oracle.Pa(z, a, thr, naive=True) - y).max() < 1e-11        # both DFT paths


def test_Pa_small_modulus_rule_G4(oracle):
    m = 8
    z = np.zeros((1, m, m), complex)                                         # F z = 0 everywhere
    a = np.full((1, m, m), 2.0)
    y = oracle.Pa(z, a, 1e-3)
    assert np.abs(np.fft.fft2(y, norm="ortho") - 2.0).max() < 1e-13          # Z' = a, phase 1
    # just above the threshold the true phase is used
    z[0] = np.fft.ifft2(np.full((m, m), 2e-3j), norm="ortho")
    y = oracle.Pa(z, a, 1e-3)
    assert np.abs(np.fft.fft2(y, norm="ortho") - 2.0j).max() < 1e-12


def test_probe_update_closed_forms(oracle):
    rng = np.random.default_rng(5)
    m, K, shape = 6, 9, (14, 15)
    pos = np.stack([rng.integers(0, shape[0] - m + 1, K), rng.integers(0, shape[1] - m + 1, K)], 1).astype(np.int32)
    w0, psi = _rc((m, m), 12), _rc(shape, 13)
    z = oracle.split(psi, w0, pos)
    assert np.abs(oracle.probe_update(psi, z, _rc((m, m), 14), pos) - w0).max() < 1e-12   # z = Q_{w0} psi -> w0
    z1 = _rc((1, m, m), 15)
    p1 = pos[:1]
    ref = z1[0] / psi[p1[0, 0]:p1[0, 0] + m, p1[0, 1]:p1[0, 1] + m]
    assert np.abs(oracle.probe_update(psi, z1, w0, p1) - ref).max() < 1e-12               # K = 1: w = z / T psi
    # Eq. (10) typed out
    zz = _rc((K, m, m), 16)
    r = np.arange(m)
    T = psi[pos[:, 0, None, None] + r[None, :, None], pos[:, 1, None, None] + r[None, None, :]]
    ref = (T.conj() * zz).sum(0) / (np.abs(T) ** 2).sum(0)
    assert np.abs(oracle.probe_update(psi, zz, w0, pos) - ref).max() < 1e-12
    # zero denominator keeps the old value
    keep = oracle.probe_update(np.zeros(shape, complex), zz, w0, pos)
    assert np.all(keep == w0)


def test_integer_geometry_P7(oracle):
    rng = np.random.default_rng(6)
    m, K, shape = 16, 40, (70, 93)
    pos = np.stack([rng.integers(0, shape[0] - m + 1, K), rng.integers(0, shape[1] - m + 1, K)], 1).astype(np.int32)
    cnt = oracle.cover_counts(m, pos, shape)
    assert cnt.sum() == K * m * m
    ref = np.zeros(shape, np.int32)
    for pr, pc in pos:
        ref[pr:pr + m, pc:pc + m] += 1
    assert np.array_equal(cnt, ref)
    idx = oracle.linear_index(m, pos, shape[1])
    assert idx[7, 3, 5] == (pos[7, 0] + 3) * shape[1] + pos[7, 1] + 5
    assert np.array_equal(np.bincount(idx.ravel(), minlength=shape[0] * shape[1]).reshape(shape), ref)
    for T in (8, 16, 32):
        ptr, frames = oracle.tile_lists(m, pos, shape, T)
        ntx = -(-shape[1] // T)
        assert ptr[0] == 0 and len(frames) == ptr[-1] and len(ptr) == (-(-shape[0] // T)) * ntx + 1
        for t in range(len(ptr) - 1):
            ty, tx = divmod(t, ntx)
            tile = np.zeros(shape, bool); tile[ty * T:(ty + 1) * T, tx * T:(tx + 1) * T] = True
            want = [i for i, (pr, pc) in enumerate(pos) if tile[pr:pr + m, pc:pc + m].any()]
            assert list(frames[ptr[t]:ptr[t + 1]]) == want          # ascending, none missing, none extra
