"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times (persistent grids of one
CTA or cluster per SM slot, many rounds, ragged last round).

config 2 (2,500 frames 128x128): one teacher-forced RAAR iteration of the whole scan against the oracle, all frames.
config 4 size (10,000 frames 256x256): the oracle cannot run the whole scan, so the frame-local operators are
compared on sampled frames the oracle computes one by one (F, F*, P_a), plus Parseval over all frames; the overlap
is compared on sampled object pixels by brute force over the frame list.
config 4 and config 5 size with the factored state in use (test_fullsize_teacher_forced_step): one RAAR iteration
from a generic state; on sampled frames the oracle's P_a and the RAAR formula evaluated in double from single
frames and the object tiles under them; the two object arrays those tiles come from are themselves checked on
sampled pixels by brute force over the frame list; the three metrics against plain torch reductions."""
import numpy as np
import pytest
import torch

import paper_1602_01448_b200 as sharp
import synth

pytestmark = pytest.mark.gpu


def rel(a, b):
    a = np.asarray(a); b = np.asarray(b)
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))


def test_config2_full_one_iteration(oracle):
    cfg = synth.config(2)
    pos, shape, I, w0, obj, wt = synth.make(cfg)
    rec = sharp.Reconstruction(cfg.m, pos, shape)
    rec.set_intensities(I); rec.set_probe(w0); rec.set_object(None)
    rec.iterate(3, cfg.beta)                       # reach a generic state with the factored form in use
    z = rec.get_frames().cpu().numpy()
    rec.iterate(1, cfg.beta)
    z1 = rec.get_frames().cpu().numpy()
    a, A2, a_rms, thr = oracle.amplitudes(I)
    want = oracle.raar(z, w0, pos, shape, a, thr, cfg.beta)
    assert rel(z1, want) < 1e-5
    per_frame = np.linalg.norm((z1 - want).reshape(cfg.K, -1), axis=1) / np.linalg.norm(want.reshape(cfg.K, -1), axis=1)
    assert per_frame.max() < 5e-5, (int(per_frame.argmax()), float(per_frame.max()))
    e = rec.errors()
    we = oracle.errors(want, z, w0, pos, shape, a, thr, A2)
    assert np.allclose(e, we, rtol=1e-4), (e, we)
    rec.close()


def test_config4_size_sampled_operators(oracle):
    cfg = synth.config(4)
    pos = synth.positions(cfg)
    K, m = cfg.K, cfg.m
    rec = sharp.Reconstruction(m, pos, cfg.shape)
    g = torch.Generator(device="cuda").manual_seed(1602)
    I = torch.rand((K, m, m), device="cuda", generator=g) * 2.0
    rec.set_intensities(I)
    w = synth.true_probe(cfg)
    rec.set_probe(w)
    z = torch.view_as_complex(torch.randn((K, m, m, 2), device="cuda", generator=g))
    sample = [0, 1, 147, 148, 2500, 7777, K - 2, K - 1]
    # F and F*: sampled frames against the oracle's own FFT, Parseval on all frames
    Z = rec.op_fft2(z, -1)
    assert abs(float(torch.linalg.vector_norm(Z) / torch.linalg.vector_norm(z)) - 1) < 1e-5
    for i in sample:
        assert rel(Z[i].cpu().numpy(), oracle.fft2(z[i].cpu().numpy(), -1)) < 1e-5, i
    Zi = rec.op_fft2(Z, +1)
    assert float(torch.linalg.vector_norm(Zi - z) / torch.linalg.vector_norm(z)) < 1e-5
    del Z, Zi
    # P_a on sampled frames (amplitudes and threshold from the full intensity array)
    y = rec.op_pa(z)
    A2 = float(I.double().sum()); thr = 1e-4 * np.sqrt(A2 / (K * m * m))
    for i in sample:
        ai = np.sqrt(I[i].cpu().numpy().astype(np.float64))
        assert rel(y[i].cpu().numpy(), oracle.Pa(z[i].cpu().numpy()[None], ai[None], thr)[0]) < 1e-5, i
    del y
    # overlap on sampled object pixels: brute force over all frames that cover the pixel, ascending index
    psi = rec.op_overlap(z)
    rng = np.random.default_rng(4)
    w64 = w.astype(np.complex128)
    for _ in range(24):
        pr, pc = int(rng.integers(0, cfg.shape[0])), int(rng.integers(0, cfg.shape[1]))
        rr, cc = pr - pos[:, 0], pc - pos[:, 1]
        hit = np.nonzero((rr >= 0) & (rr < m) & (cc >= 0) & (cc < m))[0]
        if hit.size == 0:
            assert complex(psi[pr, pc]) == 0
            continue
        fv = torch.stack([z[int(i), int(rr[i]), int(cc[i])] for i in hit]).cpu().numpy().astype(np.complex128)
        wv = w64[rr[hit], cc[hit]]
        den = np.sum(np.abs(wv) ** 2)
        if den < 1e-3:
            continue                                # G5: ratio of rounding noise
        want = np.sum(np.conj(wv) * fv) / den
        assert abs(complex(psi[pr, pc]) - want) <= 2e-5 * max(abs(want), np.sqrt(np.sum(np.abs(fv) ** 2) / den) * 1e-1), (pr, pc)
    rec.close()


def test_config3_full_one_blind_iteration(oracle):
    """The blind loop at full config-3 size: RAAR step, Eq. 9, Eq. 10, Q*Q + cross rebuild and re-gather, once,
    teacher-forced from a GPU state (reading G10 order).  The probe update divides by sum |psi|^2 and psi itself is
    a ratio at weakly lit pixels, so the bar is the oracle's own sensitivity to a 1e-7 input perturbation (x10),
    floored at the operator tolerance, as in test_probe_refinement_sequence_G10."""
    cfg = synth.config(3)
    pos, shape, I, w0, obj, wt = synth.make(cfg)
    rec = sharp.Reconstruction(cfg.m, pos, shape)
    rec.set_intensities(I); rec.set_probe(w0); rec.set_object(None)
    rec.set_probe_refine(0)
    rec.iterate(2, cfg.beta)                       # fixed-probe warm-up to a generic state
    z = rec.get_frames().cpu().numpy()
    rec.set_probe_refine(1)
    rec.iterate(1, cfg.beta)
    z1 = rec.get_frames().cpu().numpy()
    w1 = rec.get_probe().cpu().numpy()
    o = oracle.Oracle(cfg.m, pos, shape, I, w0, refine_every=1)
    o.set_frames(z)
    o.it = 0
    o.iterate(1, cfg.beta)
    rng = np.random.default_rng(5)
    o2 = oracle.Oracle(cfg.m, pos, shape, I, w0, refine_every=1)
    o2.set_frames((z * (1 + 1e-7 * rng.standard_normal(z.shape))).astype(np.complex64))
    o2.iterate(1, cfg.beta)
    assert rel(z1, o.z) < 1e-5
    tol_w = max(2e-5, 10 * rel(o2.w, o.w))
    assert rel(w1, o.w) < tol_w, (rel(w1, o.w), tol_w)
    psi = rec.get_object().cpu().numpy()
    den = oracle.overlap_den(o.w, pos, shape)
    lit = den >= 1e-3 * den.max()
    want_psi = o.object()
    tol_p = max(5e-5, 10 * rel(o2.object()[lit], want_psi[lit]))
    assert rel(psi[lit], want_psi[lit]) < tol_p
    rec.close()


def _brute_force_pixels(psi, frames, w64, pos, m, shape, rng, n=24, tol=2e-5):
    """Eq. 9 at sampled object pixels: sum over every frame covering the pixel, in double, from the frame list."""
    checked = 0
    for _ in range(n):
        pr, pc = int(rng.integers(0, shape[0])), int(rng.integers(0, shape[1]))
        rr, cc = pr - pos[:, 0], pc - pos[:, 1]
        hit = np.nonzero((rr >= 0) & (rr < m) & (cc >= 0) & (cc < m))[0]
        if hit.size == 0:
            assert complex(psi[pr, pc]) == 0
            continue
        fv = torch.stack([frames[int(i), int(rr[i]), int(cc[i])] for i in hit]).cpu().numpy().astype(np.complex128)
        wv = w64[rr[hit], cc[hit]]
        den = np.sum(np.abs(wv) ** 2)
        if den < 1e-3 * float(np.sum(np.abs(w64) ** 2)) / m ** 2 * hit.size:
            continue                                # G5: ratio of rounding noise
        want = np.sum(np.conj(wv) * fv) / den
        assert abs(complex(psi[pr, pc]) - want) <= tol * max(abs(want), np.sqrt(np.sum(np.abs(fv) ** 2) / den) * 1e-1), (pr, pc)
        checked += 1
    assert checked >= n // 3


@pytest.mark.parametrize("n", [4, 5])
def test_fullsize_teacher_forced_step(oracle, n):
    """configs 4 (10,000 frames 256x256) and 5 (1,600 frames 512x512) at full size, in the launch configuration
    bench.py times (many rounds per cluster), with the factored state z = c + w T psi_v in use."""
    cfg = synth.config(n)
    pos = synth.positions(cfg)
    K, m, shape, beta = cfg.K, cfg.m, cfg.shape, cfg.beta
    rec = sharp.Reconstruction(m, pos, shape)
    g = torch.Generator(device="cuda").manual_seed(1602 + n)
    w = synth.true_probe(cfg)
    # intensities of the right scale: |F(w x random-phase object)|^2-like level, random
    I = torch.rand((K, m, m), device="cuda", generator=g) * float(2.0 * np.sum(np.abs(w) ** 2) / m ** 2)
    rec.set_intensities(I)
    rec.set_probe(w)
    rec.set_object(None)
    rec.iterate(2, beta)                               # generic state, psi_v != 0
    z = rec.get_frames()
    psi_z = rec.get_object()
    y = rec.op_pa(z)
    e0 = rec.errors()
    rec.iterate(1, beta)
    z1 = rec.get_frames()
    psi_y = rec.get_object()
    e1 = rec.errors()
    w64 = w.astype(np.complex128)
    A2 = float(I.double().sum()); thr = 1e-4 * np.sqrt(A2 / (K * m * m))
    rng = np.random.default_rng(40 + n)
    # the two object arrays, Eq. 9 by brute force on sampled pixels: psi_z = L z, psi_y = L y (= L z', identity O7)
    _brute_force_pixels(psi_z, z, w64, pos, m, shape, rng)
    _brute_force_pixels(psi_y, y, w64, pos, m, shape, rng)
    _brute_force_pixels(psi_y, z1, w64, pos, m, shape, rng, tol=5e-5)
    # sampled frames: P_a by the oracle, then step 5 (reading G1) typed out in double from the tiles
    pz, py = psi_z.cpu().numpy().astype(np.complex128), psi_y.cpu().numpy().astype(np.complex128)
    for i in [0, 1, K // 3, K // 2 + 1, K - 2, K - 1]:
        zi = z[i].cpu().numpy()
        ai = np.sqrt(np.maximum(I[i].cpu().numpy().astype(np.float64), 0))
        yi = oracle.Pa(zi[None], ai[None], thr)[0]
        assert rel(y[i].cpu().numpy(), yi) < 1e-5, i
        r, c = int(pos[i, 0]), int(pos[i, 1])
        want = 2 * beta * w64 * py[r:r + m, c:c + m] + (1 - 2 * beta) * yi + beta * (zi - w64 * pz[r:r + m, c:c + m])
        assert rel(z1[i].cpu().numpy(), want) < 2e-5, (i, rel(z1[i].cpu().numpy(), want))
    # the metrics at both states against plain torch reductions over all frames (double accumulation)
    wt_ = torch.from_numpy(w).cuda()

    def eps_q(zz, psi):
        s = 0.0
        for i in range(K):
            r, c = int(pos[i, 0]), int(pos[i, 1])
            s += float(torch.sum(torch.abs(wt_ * psi[r:r + m, c:c + m] - zz[i]).double() ** 2))
        return np.sqrt(s / A2)

    ea0 = float(torch.sqrt(torch.sum(torch.abs(y - z).double() ** 2) / A2))
    assert abs(e0[0] / ea0 - 1) < 1e-4 and abs(e0[1] / eps_q(z, psi_z) - 1) < 1e-4, (e0, ea0)
    y1 = rec.op_pa(z1)
    ea1 = float(torch.sqrt(torch.sum(torch.abs(y1 - z1).double() ** 2) / A2))
    ed1 = float(torch.sqrt(torch.sum(torch.abs(z1 - z).double() ** 2) / A2))
    assert abs(e1[0] / ea1 - 1) < 1e-4 and abs(e1[2] / ed1 - 1) < 1e-4, (e1, ea1, ed1)
    assert abs(e1[1] / eps_q(z1, psi_y) - 1) < 1e-4
    rec.close()


@pytest.mark.parametrize("cfgno", [2, 3])
def test_fullsize_runs_are_bitwise_reproducible_under_the_dynamic_schedule(cfgno):
    """m = 128 at full size: frames after the first are handed to the CTAs by a global counter and the CTAs start in
    phases, so which CTA transforms which frame differs from run to run.  The result must not: three runs, the third on a
    different persistent grid, give bit-identical frames, illumination and residuals (no float atomics, fixed summation
    orders; the residual pass keeps the fixed round-robin)."""
    cfg = synth.config(cfgno)
    pos, shape, I, w0, obj, wt = synth.make(cfg)
    ref = None
    for run in range(3):
        rec = sharp.Reconstruction(cfg.m, pos, shape)
        if run == 2:
            rec.set_frame_slots(37)
        rec.set_probe_refine(cfg.refine_every)
        rec.set_intensities(I); rec.set_probe(w0); rec.set_object(None)
        rec.iterate(12, cfg.beta)
        got = (rec.get_frames(), rec.get_probe(), rec.get_object())
        e = rec.errors()
        torch.cuda.synchronize()
        if ref is None:
            ref, ref_e = tuple(t.clone() for t in got), e
        else:
            assert all(torch.equal(a, b) for a, b in zip(got, ref)), run
            if run == 1:
                assert np.array_equal(e, ref_e)
            else:
                assert np.allclose(e, ref_e, rtol=1e-6)      # other grid: the per-CTA partial sums group other frames
        rec.close()
