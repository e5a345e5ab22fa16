"""Pins for the oracle functions of SURVEY.md section 8(f): eps_0 (Eq. 14), the default initialisations (steps 2-3),
the illumination constraints and re-centring (step 7), and the periodic T_i of the Fig. 3 simulation.

Every expected value here comes from numpy written out independently of oracle/ (fancy indexing, numpy's FFT,
np.roll, Python integers) or from a closed form; none is the oracle's own formula re-typed around its own helpers.
"""
import numpy as np
import pytest

from oracle import sharp_oracle as orc

RNG = np.random.default_rng(20260211)


def crandn(*s):
    return RNG.standard_normal(s) + 1j * RNG.standard_normal(s)


def np_overlap_num(f, w, pos, shape, periodic=False):
    """sum_i conj(w) f_i scattered with np.add.at (independent of oracle/)."""
    K, m, _ = f.shape
    num = np.zeros(shape, complex)
    r = np.arange(m)
    for i in range(K):
        rows = pos[i, 0] + r
        cols = pos[i, 1] + r
        if periodic:
            rows, cols = rows % shape[0], cols % shape[1]
        np.add.at(num, (rows[:, None], cols[None, :]), np.conj(w) * f[i])
    return num


def small_scan(m=8, n=20, K=9):
    pos = RNG.integers(0, n - m + 1, size=(K, 2)).astype(np.int32)
    return m, (n, n + 3), pos, crandn(m, m), crandn(n, n + 3)


# ---- eps_0 -------------------------------------------------------------------------------------------------------
def test_eps0_is_the_minimum_over_phi_brute_force():
    m, shape, pos, w, psi0 = small_scan()
    z = crandn(len(pos), m, m)
    e, phi = orc.eps0(z, psi0, w, pos, shape, return_phi=True)
    A = np_overlap_num(z, w, pos, shape)
    z0 = np.stack([w * psi0[p[0]:p[0] + m, p[1]:p[1] + m] for p in pos])
    B = np_overlap_num(z0, w, pos, shape)
    phis = np.linspace(-np.pi, np.pi, 20001)
    scan = np.array([np.linalg.norm(np.exp(1j * t) * A - B) for t in phis]) / np.linalg.norm(B)
    assert e <= scan.min() + 1e-12                     # nothing on the grid is below it
    assert abs(e - scan.min()) < 1e-6                  # and the grid gets that close (step 3e-4 rad, quadratic minimum)
    assert abs(np.angle(np.exp(1j * (phi - phis[scan.argmin()])))) < 4e-4
    # expanded closed form ||A||^2 + ||B||^2 - 2 |<B,A>|
    cf = np.sqrt(np.vdot(A, A).real + np.vdot(B, B).real - 2 * abs(np.vdot(B, A))) / np.linalg.norm(B)
    assert abs(e - cf) < 1e-12


def test_eps0_zero_at_the_solution_up_to_a_global_phase_and_phase_invariant():
    m, shape, pos, w, psi0 = small_scan()
    z0 = orc.split(psi0, w, pos)
    e, phi = orc.eps0(np.exp(0.7j) * z0, psi0, w, pos, shape, return_phi=True)
    assert e < 1e-14 and abs(phi + 0.7) < 1e-12
    z = z0 + 0.1 * crandn(*z0.shape)
    e1 = orc.eps0(z, psi0, w, pos, shape)
    e2 = orc.eps0(np.exp(-2.1j) * z, psi0, w, pos, shape)
    assert e1 > 1e-3 and abs(e1 - e2) < 1e-13


def test_eps0_uses_the_overlap_sum_not_the_frames_and_a_separate_w0():
    m, shape, pos, w, psi0 = small_scan()
    z = crandn(len(pos), m, m)
    # a perturbation in the null space of Q* (orthogonal to the range of Q) must not change eps_0
    y = crandn(len(pos), m, m)
    y_null = y - orc.PQ(y, w, pos, shape)
    assert abs(orc.eps0(z, psi0, w, pos, shape) - orc.eps0(z + y_null, psi0, w, pos, shape)) < 1e-12
    # z0 formed with the solution's own illumination w0
    w0 = crandn(m, m)
    z0 = np.stack([w0 * psi0[p[0]:p[0] + m, p[1]:p[1] + m] for p in pos])
    A, B = np_overlap_num(z, w, pos, shape), np_overlap_num(z0, w, pos, shape)
    cf = np.sqrt(np.vdot(A, A).real + np.vdot(B, B).real - 2 * abs(np.vdot(B, A))) / np.linalg.norm(B)
    assert abs(orc.eps0(z, psi0, w, pos, shape, w0=w0) - cf) < 1e-12


# ---- default initialisations -------------------------------------------------------------------------------------
def test_default_probe_is_ifft_of_sqrt_mean_frame_at_the_frame_centre():
    K, m = 5, 16
    I = (RNG.random((K, m, m)) * 3).astype(np.float32)
    I[0, 2, 3] = -4.0                                   # clamped (G14)
    ref = np.fft.fftshift(np.fft.ifft2(np.sqrt(np.maximum(I.astype(float), 0).mean(axis=0)), norm="ortho"))
    assert np.abs(orc.default_probe(I) - ref).max() < 1e-12


def test_default_probe_recovers_a_zero_phase_pupil_probe_exactly():
    """Flat object and a probe whose pupil is real and non-negative: every frame is |F w|^2, so F* sqrt(mean I) is the
    probe itself, peak at the frame centre (closed-form special case; pins the shift and the unitary scale)."""
    m, K = 32, 4
    u = np.arange(m) - m // 2
    D = ((u[:, None] ** 2 + u[None, :] ** 2) <= 36).astype(float)
    w = np.fft.fftshift(np.fft.ifft2(np.fft.ifftshift(D), norm="ortho"))
    I = np.repeat((np.abs(np.fft.fft2(w, norm="ortho")) ** 2)[None], K, axis=0)
    w0 = orc.default_probe(I.astype(np.float32))
    assert np.abs(w0 - w).max() < 1e-6                   # float32 intensities
    assert np.unravel_index(np.abs(w0).argmax(), w0.shape) == (m // 2, m // 2)


def py_splitmix64(x):
    M = (1 << 64) - 1
    x = (x + 0x9E3779B97F4A7C15) & M
    z = x
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & M
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & M
    return z ^ (z >> 31)


def test_random_object_is_the_documented_counter_based_draw():
    seed, shape = 1602014480, (7, 11)
    psi = orc.random_object(shape, seed)
    k = py_splitmix64(seed)
    ref = np.array([(py_splitmix64((k + p) & ((1 << 64) - 1)) >> 40) / 16777216.0 for p in range(77)]).reshape(shape)
    assert np.array_equal(psi.real, ref.astype(np.float32).astype(float)) and not psi.imag.any()
    big = orc.random_object((200, 200), seed + 1).real
    assert big.min() >= 0.0 and big.max() < 1.0 and abs(big.mean() - 0.5) < 0.01 and abs(big.var() - 1 / 12) < 0.005
    assert not np.array_equal(orc.random_object(shape, seed + 1), psi)


# ---- illumination constraints --------------------------------------------------------------------------------------
def test_probe_mask_projection():
    m = 16
    w = crandn(m, m)
    mask = (RNG.random((m, m)) < 0.4).astype(float)
    out = orc.probe_mask(w, mask)
    assert np.abs(np.fft.fft2(out, norm="ortho") - np.fft.fft2(w, norm="ortho") * mask).max() < 1e-12
    assert np.abs(orc.probe_mask(out, mask) - out).max() < 1e-13          # idempotent for a 0/1 support
    assert np.abs(orc.probe_mask(w, np.ones((m, m))) - w).max() < 1e-13   # full support: identity
    # mask indexed like the transform (DC at [0,0]): keeping only DC leaves the mean
    dc = np.zeros((m, m)); dc[0, 0] = 1
    assert np.abs(orc.probe_mask(w, dc) - w.mean()).max() < 1e-13


def test_probe_amplitude_projection():
    m = 16
    w = crandn(m, m)
    aw = RNG.random((m, m)) + 0.1
    out = orc.probe_amplitude(w, aw)
    W, O = np.fft.fft2(w, norm="ortho"), np.fft.fft2(out, norm="ortho")
    assert np.abs(np.abs(O) - aw).max() < 1e-12                            # |F w'| = a_w
    assert np.abs(O / np.abs(O) - W / np.abs(W)).max() < 1e-12             # phases kept
    assert np.abs(orc.probe_amplitude(out, aw) - out).max() < 1e-12        # idempotent
    assert np.abs(orc.probe_amplitude(w, np.abs(W)) - w).max() < 1e-12     # a_w = |F w|: identity
    # G24: a coefficient below the threshold takes phase 1
    w1 = np.full((m, m), 1.0 + 0j)                                          # F w1 = m at DC, 0 elsewhere
    O1 = np.fft.fft2(orc.probe_amplitude(w1, aw), norm="ortho")
    assert np.abs(O1 - aw).max() < 1e-12


def test_probe_recentre_moves_a_displaced_probe_back_by_the_known_integer():
    m = 64
    r = np.arange(m)
    g = lambda cr, cc: np.exp(-((r[:, None] - cr) ** 2 + (r[None, :] - cc) ** 2) / (2 * 4.0 ** 2)) * np.exp(0.3j * r[None, :])
    w = g(m // 2 + 3, m // 2 - 5)
    out, d = orc.probe_recentre(w)
    assert d == (-3, 5)
    assert np.array_equal(out, np.roll(w, d, axis=(0, 1)))
    out2, d2 = orc.probe_recentre(out)
    assert d2 == (0, 0) and np.array_equal(out2, out)
    # the mass is |w|^2, not |w|: two points, amplitude 1 at row 10 and 3 at row 40 -> cm = (10 + 9*40)/10 = 37 (|w|: 32.5)
    w = np.zeros((m, m), complex); w[10, 32] = 1; w[40, 32] = 3
    assert orc.probe_recentre(w)[1] == (32 - 37, 0)
    # rounding: cm = 31.4 -> d = round(0.6) = 1 ; cm = 31.6 -> d = round(0.4) = 0
    w = np.zeros((m, m), complex); w[31, 32] = np.sqrt(0.6); w[32, 32] = np.sqrt(0.4)
    assert orc.probe_recentre(w)[1] == (1, 0)
    w[31, 32], w[32, 32] = np.sqrt(0.4), np.sqrt(0.6)
    assert orc.probe_recentre(w)[1] == (0, 0)
    z = np.zeros((m, m), complex)
    assert orc.probe_recentre(z)[1] == (0, 0)


def test_oracle_sequence_with_constraints_follows_step_7_order():
    m, n = 8, 20
    pos = np.array([[0, 0], [0, 6], [6, 0], [6, 6], [3, 3], [12, 12], [12, 5], [5, 12]], np.int32)
    psi, w = crandn(n, n), crandn(m, m)
    I = (np.abs(np.fft.fft2(orc.split(psi, w, pos), norm="ortho")) ** 2).astype(np.float32)
    w_start = (w + 0.3 * crandn(m, m)).astype(np.complex64)
    aw = np.abs(np.fft.fft2(w, norm="ortho"))
    for kw in (dict(probe_mask=(aw > 0.5).astype(float)), dict(probe_amplitude=aw), dict()):
        o = orc.Oracle(m, pos, (n, n), I, w_start, refine_every=1, recentre=True, **kw)
        o.iterate(1, 0.75)
        a, A2, a_rms, thr = orc.amplitudes(I)
        w64 = w_start.astype(complex)
        z1 = orc.raar(orc.split(np.ones((n, n)), w64, pos), w64, pos, (n, n), a, thr, 0.75)
        w1 = orc.probe_update(orc.L(z1, w64, pos, (n, n)), z1, w64, pos)
        if "probe_mask" in kw:
            w1 = orc.probe_mask(w1, kw["probe_mask"])
        elif "probe_amplitude" in kw:
            w1 = orc.probe_amplitude(w1, aw)
        w1, d = orc.probe_recentre(w1)
        assert np.array_equal(o.w, w1) and o.shifts == [d] and np.array_equal(o.z, z1)


# ---- periodic T_i (Fig. 3 simulation) --------------------------------------------------------------------------------
def test_periodic_split_overlap_and_integer_artefacts():
    m, shape = 8, (20, 23)
    pos = np.array([[0, 0], [15, 19], [19, 22], [7, 18], [16, 3], [12, 15]], np.int32)    # several wrap
    psi, w = crandn(*shape), crandn(m, m)
    z = orc.split(psi, w, pos)
    for i, (pr, pc) in enumerate(pos):
        assert np.abs(z[i] - w * np.roll(psi, (-pr, -pc), axis=(0, 1))[:m, :m]).max() < 1e-14
    f = crandn(len(pos), m, m)
    num = orc.overlap_num(f, w, pos, shape)
    assert np.abs(num - np_overlap_num(f, w, pos, shape, periodic=True)).max() < 1e-12
    assert abs(np.vdot(z, f) - np.vdot(psi, num)) < 1e-10 * abs(np.vdot(z, f))            # <Q psi, f> = <psi, Q* f>
    cnt = orc.cover_counts(m, pos, shape)
    assert cnt.sum() == len(pos) * m * m
    ref = np.zeros(shape, int)
    r = np.arange(m)
    for pr, pc in pos:
        ref[np.ix_((pr + r) % shape[0], (pc + r) % shape[1])] += 1
    assert np.array_equal(cnt, ref)
    idx = orc.linear_index_periodic(m, pos, shape)
    assert np.array_equal(idx, ((pos[:, 0, None, None] + r[None, :, None]) % shape[0]) * shape[1]
                          + (pos[:, 1, None, None] + r[None, None, :]) % shape[1])
    T = 4
    ptr, frames = orc.tile_lists_periodic(m, pos, shape, T)
    tiles_c = (shape[1] + T - 1) // T
    for t in range(len(ptr) - 1):
        ty, tx = divmod(t, tiles_c)
        want = [i for i in range(len(pos)) if ref_hits(ref_cover(m, pos[i], shape), ty, tx, T)]
        assert list(frames[ptr[t]:ptr[t + 1]]) == want


def ref_cover(m, p, shape):
    c = np.zeros(shape, bool)
    r = np.arange(m)
    c[np.ix_((p[0] + r) % shape[0], (p[1] + r) % shape[1])] = True
    return c


def ref_hits(cover, ty, tx, T):
    return bool(cover[ty * T:(ty + 1) * T, tx * T:(tx + 1) * T].any())


def test_periodic_lists_equal_the_plain_ones_when_nothing_wraps():
    m, shape = 8, (30, 30)
    pos = RNG.integers(0, 30 - m + 1, size=(12, 2)).astype(np.int32)
    p0, f0 = orc.tile_lists(m, pos, shape, 8)
    p1, f1 = orc.tile_lists_periodic(m, pos, shape, 8)
    assert np.array_equal(p0, p1) and np.array_equal(f0, f1)
    assert np.array_equal(orc.linear_index(m, pos, shape[1]), orc.linear_index_periodic(m, pos, shape))


def test_fixed_point_with_periodic_boundary():
    """RAAR's fixed point (P4) on a periodic scan: every object pixel is covered, frames wrap."""
    m, n = 8, 16
    pos = np.array([[r, c] for r in range(0, n, 4) for c in range(0, n, 4)], np.int32)      # 16 frames, all wrap classes
    psi, w = crandn(n, n), crandn(m, m)
    z0 = orc.split(psi, w, pos)
    a = np.abs(np.fft.fft2(z0, norm="ortho"))
    z1 = orc.raar(z0, w, pos, (n, n), a, 0.0, 0.75)
    assert np.abs(z1 - z0).max() < 1e-12
    assert (orc.cover_counts(m, pos, (n, n)) == 4).all()
