"""The seeded input generator (paper_1602_01448_b200/synth.py): reproducible, in range, and the sizes of
BASELINE.json's configs as read in SURVEY.md section 8(d)."""
import numpy as np

import synth


def test_config_shapes_and_counts():
    want = {1: (64, 100, (208, 208)), 2: (128, 2500, (1704, 1704)), 3: (128, 2500, (1704, 1704)),
            4: (256, 10000, (5020, 5020)), 5: (512, 1600, (4352, 4352))}
    for n, (m, K, shape) in want.items():
        cfg = synth.config(n)
        assert (cfg.m, cfg.K, cfg.shape) == (m, K, shape)
        pos = synth.positions(cfg)
        assert pos.dtype == np.int32 and pos.shape == (K, 2)
        assert pos.min() >= 0 and pos[:, 0].max() <= shape[0] - m and pos[:, 1].max() <= shape[1] - m


def test_counter_based_and_reproducible():
    u1 = synth.uniform(7, 3, np.arange(1000))
    u2 = synth.uniform(7, 3, np.arange(500, 1000))
    assert np.array_equal(u1[500:], u2) and 0.0 <= u1.min() and u1.max() < 1.0
    assert abs(u1.mean() - 0.5) < 0.05 and not np.array_equal(u1, synth.uniform(7, 4, np.arange(1000)))
    lam = np.full(20000, 3.7)
    k = synth.poisson(lam, 1, 2)
    assert abs(k.mean() - 3.7) < 0.1 and abs(k.var() - 3.7) < 0.3
    kb = synth.poisson(np.full(20000, 400.0), 1, 2)
    assert abs(kb.mean() - 400) < 1.0 and abs(kb.var() - 400) < 30


def test_tiny_scan_recipe():
    cfg = synth.config(1)
    pos, shape, I, w0, obj, wt = synth.make(cfg)
    assert I.dtype == np.float32 and I.shape == (100, 64, 64) and w0.dtype == np.complex64
    assert abs((np.abs(wt.astype(complex)) ** 2).sum() - 441) < 1e-3          # pupil pixels with rho <= 12
    assert np.abs(obj).min() >= 0.8 - 1e-6 and np.abs(obj).max() <= 1 + 1e-6
    assert np.abs(np.angle(obj)).max() <= np.pi / 2 + 1e-6
    # Parseval: mean photons per frame * (1/s) = mean sum|z|^2 ; Poisson scale 1e4 photons/frame
    s = 1e4 / synth.intensities(synth.reduced(cfg, 10, photons=0.0)).reshape(100, -1).sum(1).mean()
    counts = I.astype(np.float64) * s
    assert np.abs(counts - np.rint(counts)).max() < 1e-2 and abs(counts.reshape(100, -1).sum(1).mean() - 1e4) < 300
    assert np.array_equal(I, synth.make(cfg)[2])
    # probe sits at the frame centre, diffraction DC at index [0,0] (G19)
    r, c = np.unravel_index(np.argmax(np.abs(wt)), wt.shape)
    assert abs(r - 32) <= 1 and abs(c - 32) <= 1
    u = np.minimum(np.arange(64), 64 - np.arange(64))
    disc = (u[:, None] ** 2 + u[None, :] ** 2) <= 12 ** 2
    tot = I.sum(0)
    # the i.i.d. random object scatters ~half of the photons outside the pupil disc, so the contrast is ~7x, not >>1
    assert tot[disc].mean() > 4 * tot[~disc].mean()
