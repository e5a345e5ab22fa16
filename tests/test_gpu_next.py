"""GPU parity for the rows of SURVEY.md section 8(f): eps_0 (Eq. 14), the default initialisations (steps 2-3), the
illumination constraints and re-centring (step 7).  Everything goes through the C ABI and is compared with the oracle
on the same seeded inputs: floats at rel-L2 <= 1e-5 (operators) / 1e-4 (metrics), integers (random draw, shifts)
exactly."""
import dataclasses

import numpy as np
import pytest

import paper_1602_01448_b200 as sharp
import synth

pytestmark = pytest.mark.gpu

OP_TOL = 1e-5
EPS_TOL = 1e-4


def rel(a, b):
    a = np.asarray(a); b = np.asarray(b)
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))


def _rc(shape, seed, scale=1.0):
    rng = np.random.default_rng(seed)
    return ((rng.standard_normal(shape) + 1j * rng.standard_normal(shape)) * scale).astype(np.complex64)


SCANS = {"m64": (1, 6), "m128": (3, 5), "m256": (4, 4), "m512": (5, 7)}


@pytest.fixture(scope="module", params=list(SCANS), ids=list(SCANS))
def scan(request):
    n, grid = SCANS[request.param]
    cfg = synth.reduced(synth.config(n), grid)
    if cfg.kind == "fermat":
        cfg = dataclasses.replace(cfg, step=20)
    pos, shape, I, w0, obj, wt = synth.make(cfg)
    rec = sharp.Reconstruction(cfg.m, pos, shape)
    rec.set_intensities(I)
    rec.set_probe(wt)
    yield dict(cfg=cfg, pos=pos, shape=shape, I=I, w0=w0, obj=obj, wt=wt, rec=rec)
    rec.close()


# ---- eps_0 -------------------------------------------------------------------------------------------------------
def test_eps0_against_the_oracle(scan, oracle):
    cfg, rec = scan["cfg"], scan["rec"]
    rec.set_probe(scan["wt"])
    z = synth.exit_waves(cfg, scan["obj"], scan["wt"], scan["pos"]).astype(np.complex64)
    for k, noise in enumerate((0.3, 1e-2, 1e-4)):
        zn = (np.exp(0.9j) * z * (1 + noise * _rc(z.shape, 40 + k))).astype(np.complex64)
        rec.set_frames(zn)
        got = rec.eps0(scan["obj"])
        want = oracle.eps0(zn, scan["obj"], scan["wt"], scan["pos"], scan["shape"])
        assert abs(got - want) <= EPS_TOL * want + 2e-7, (noise, got, want)
    # exactly at the solution, up to the global phase: the fp32 floor
    rec.set_frames((np.exp(-2.0j) * z).astype(np.complex64))
    assert rec.eps0(scan["obj"]) < 1e-6


def test_eps0_with_the_solutions_own_illumination_and_after_iterations(scan, oracle):
    cfg, rec = scan["cfg"], scan["rec"]
    w_run = (scan["wt"] * (1 + 0.2 * _rc(scan["wt"].shape, 51))).astype(np.complex64)
    rec.set_probe(w_run)
    rec.set_object(None)
    rec.iterate(3, cfg.beta)
    o = oracle.Oracle(cfg.m, scan["pos"], scan["shape"], scan["I"], w_run)
    o.set_frames(rec.get_frames().cpu().numpy())          # eps_0 is a function of the state: evaluate both at the same z
    got = rec.eps0(scan["obj"], scan["wt"])
    want = o.eps0(scan["obj"], w0=scan["wt"])
    assert abs(got - want) <= EPS_TOL * want, (got, want)
    got2, want2 = rec.eps0(scan["obj"]), o.eps0(scan["obj"])
    assert abs(got2 - want2) <= EPS_TOL * want2
    # non-mutating: the frames and residuals are unchanged by the evaluation
    assert rel(rec.get_frames().cpu().numpy(), o.z) < 1e-7
    rec.set_probe(scan["wt"])


# ---- default initialisations -------------------------------------------------------------------------------------
def test_random_object_bit_exact_and_its_frames(scan, oracle):
    cfg, rec = scan["cfg"], scan["rec"]
    seed = 1602014480 + cfg.m
    want = oracle.random_object(scan["shape"], seed)
    got = rec.op_random_object(seed).cpu().numpy()
    assert np.array_equal(got.real, want.real.astype(np.float32)) and not got.imag.any()
    rec.set_probe(scan["wt"])
    rec.init_object_random(seed)
    z = rec.get_frames().cpu().numpy()
    assert rel(z, oracle.split(want, scan["wt"], scan["pos"])) < OP_TOL
    o = oracle.Oracle(cfg.m, scan["pos"], scan["shape"], scan["I"], scan["wt"], psi0=want)
    rec.iterate(2, cfg.beta)
    o.iterate(2, cfg.beta)
    assert rel(rec.get_frames().cpu().numpy(), o.z) < 3e-5
    assert np.allclose(rec.errors(), o.errors(), rtol=EPS_TOL)


def test_default_probe(scan, oracle):
    cfg, rec = scan["cfg"], scan["rec"]
    rec.init_probe()
    got = rec.get_probe().cpu().numpy()
    want = oracle.default_probe(scan["I"])
    assert rel(got, want) < OP_TOL
    # it is installed like sharp_set_probe: Q*Q follows
    f = _rc((cfg.K, cfg.m, cfg.m), 61)
    den = oracle.overlap_den(want, scan["pos"], scan["shape"])
    lit = den >= 1e-3 * den.max()
    assert rel(rec.op_overlap(f).cpu().numpy()[lit], oracle.L(f, want, scan["pos"], scan["shape"])[lit]) < OP_TOL
    rec.set_probe(scan["wt"])


# ---- illumination constraints --------------------------------------------------------------------------------------
def _constraints(scan):
    m = scan["cfg"].m
    aw = np.abs(np.fft.fft2(scan["wt"].astype(np.complex128), norm="ortho"))
    mask = (aw > 1e-3 * aw.max()).astype(np.float32)
    return mask, aw.astype(np.float32)


@pytest.mark.parametrize("kind", ["mask", "amplitude", "none"])
@pytest.mark.parametrize("recentre", [False, True])
def test_op_probe_constrain(scan, oracle, kind, recentre):
    cfg, rec = scan["cfg"], scan["rec"]
    m = cfg.m
    mask, aw = _constraints(scan)
    w = np.roll(scan["wt"] * (1 + 0.2 * _rc((m, m), 71)), (5, -9), axis=(0, 1)).astype(np.complex64)
    rec.set_probe_constraint(kind, {"mask": mask, "amplitude": aw, "none": None}[kind])
    rec.set_probe_recentre(recentre)
    got = rec.op_probe_constrain(w).cpu().numpy()
    want = w.astype(np.complex128)
    if kind == "mask":
        want = oracle.probe_mask(want, mask)
    elif kind == "amplitude":
        want = oracle.probe_amplitude(want, aw)
    if recentre:
        want, d = oracle.probe_recentre(want)
        assert rec.get_probe_shift()[0] == d and d != (0, 0)
    assert rel(got, want) < OP_TOL
    if kind == "amplitude":
        assert rel(np.abs(np.fft.fft2(got.astype(np.complex128), norm="ortho")), aw) < OP_TOL
    rec.set_probe_constraint("none")
    rec.set_probe_recentre(False)


@pytest.mark.parametrize("kind", ["mask", "amplitude"])
def test_blind_sequence_with_constraints_step_7(scan, oracle, kind):
    """Three blind iterations with the constraint and the re-centring on, teacher-forced after each: both sides start
    every iteration from the GPU's frames and illumination and must agree on z', w' and the integer shift."""
    cfg, rec = scan["cfg"], scan["rec"]
    m = cfg.m
    mask, aw = _constraints(scan)
    con = mask if kind == "mask" else aw
    w_start = np.roll(scan["w0"], (3, -2), axis=(0, 1)).astype(np.complex64)       # off-centre: the first shift is not 0
    rec.set_probe(w_start)
    rec.set_probe_refine(1)
    rec.set_probe_constraint(kind, con)
    rec.set_probe_recentre(True)
    # start from noisy exit waves, not from the flat object: with a Gaussian probe |F z0| falls smoothly through the G4
    # threshold and single pixels there take different branches in fp32 and fp64 ("Parity unpinned")
    z = (synth.exit_waves(cfg, scan["obj"], w_start, scan["pos"]) * (1 + 0.2 * _rc((cfg.K, m, m), 72))).astype(np.complex64)
    rec.set_frames(z)
    w = w_start
    total = np.zeros(2, int)
    for it in range(3):
        o = oracle.Oracle(m, scan["pos"], scan["shape"], scan["I"], w, refine_every=1, recentre=True,
                          **({"probe_mask": mask} if kind == "mask" else {"probe_amplitude": aw}))
        o.set_frames(z)
        o.iterate(1, cfg.beta)
        rec.iterate(1, cfg.beta)
        z = rec.get_frames().cpu().numpy()
        w = rec.get_probe().cpu().numpy()
        last, tot = rec.get_probe_shift()
        total += np.array(o.shifts[0])
        assert last == o.shifts[0] and tot == tuple(total), (it, last, o.shifts, tot)
        assert rel(z, o.z) < OP_TOL, it
        assert rel(w, o.w) < 3e-5, it
        den = oracle.overlap_den(o.w, scan["pos"], scan["shape"])
        lit = den >= 1e-3 * den.max()
        assert rel(rec.get_object().cpu().numpy()[lit], o.object()[lit]) < 3e-5
    rec.set_probe_refine(0)
    rec.set_probe_constraint("none")
    rec.set_probe_recentre(False)
    rec.set_probe(scan["wt"])


# ---- periodic boundary (the Fig. 3 simulation) -----------------------------------
def _periodic_cfg(m):
    """The Fig. 3 recipe (dense raster on a torus, exact illumination, noise-free) at sizes the oracle affords: the image
    is grid * step pixels, at least m + 31, and most frames wrap around an edge."""
    grid, step = {64: (12, 8), 128: (10, 16), 256: (6, 48), 512: (3, 184)}[m]
    base = synth.config(6)
    return dataclasses.replace(base, m=m, grid=grid, step=step, periodic=grid * step, pupil_radius=12.0 * m / 64,
                               name=f"fig3-m{m}")


@pytest.fixture(scope="module", params=[(64, 0), (64, 7), (128, 0), (128, 9), (256, 5), (512, 2)],
                ids=lambda p: f"m{p[0]}-slots{p[1]}")
def pscan(request):
    m, slots = request.param
    cfg = _periodic_cfg(m)
    pos, shape, I, w0, obj, wt = synth.make(cfg)
    assert ((pos[:, 0] + m > shape[0]) | (pos[:, 1] + m > shape[1])).sum() > len(pos) // 3
    rec = sharp.Reconstruction(m, pos, shape, periodic=True)
    if slots:
        rec.set_frame_slots(slots)
    rec.set_intensities(I)
    rec.set_probe(wt)
    yield dict(cfg=cfg, pos=pos, shape=shape, I=I, obj=obj, wt=wt, rec=rec)
    rec.close()


def test_periodic_frame_index_bit_exact(pscan, oracle):
    idx = pscan["rec"].frame_index().cpu().numpy()
    assert np.array_equal(idx, oracle.linear_index_periodic(pscan["cfg"].m, pscan["pos"], pscan["shape"]))


def test_periodic_operators(pscan, oracle):
    cfg, rec = pscan["cfg"], pscan["rec"]
    psi = _rc(pscan["shape"], 81)
    assert rel(rec.op_split(psi).cpu().numpy(), oracle.split(psi, pscan["wt"], pscan["pos"])) < OP_TOL
    f = _rc((cfg.K, cfg.m, cfg.m), 82)
    got = rec.op_overlap(f).cpu().numpy()
    want = oracle.L(f, pscan["wt"], pscan["pos"], pscan["shape"])
    den = oracle.overlap_den(pscan["wt"], pscan["pos"], pscan["shape"])
    lit = den >= 1e-3 * den.max()
    assert rel(got[lit], want[lit]) < OP_TOL and rel(got * np.sqrt(den), want * np.sqrt(den)) < OP_TOL
    z = (synth.exit_waves(cfg, pscan["obj"], pscan["wt"], pscan["pos"]) * (1 + 0.3 * _rc(f.shape, 83))).astype(np.complex64)
    assert rel(rec.op_probe(psi, z).cpu().numpy(), oracle.probe_update(psi, z, pscan["wt"], pscan["pos"])) < OP_TOL


@pytest.mark.parametrize("beta", [0.75, 0.9])
def test_periodic_raar_steps_errors_eps0(pscan, oracle, beta):
    cfg, rec = pscan["cfg"], pscan["rec"]
    z0 = (synth.exit_waves(cfg, pscan["obj"], pscan["wt"], pscan["pos"]) * (1 + 0.2 * _rc((cfg.K, cfg.m, cfg.m), 84))).astype(np.complex64)
    rec.set_probe(pscan["wt"])
    rec.set_frames(z0)
    o = oracle.Oracle(cfg.m, pscan["pos"], pscan["shape"], pscan["I"], pscan["wt"])
    o.set_frames(z0)
    for step in range(2):                                  # the second step runs on the factored state (psi_v gather with wrap)
        rec.iterate(1, beta)
        o.iterate(1, beta)
        assert rel(rec.get_frames().cpu().numpy(), o.z) < (OP_TOL if step == 0 else 3e-5)
        assert np.allclose(rec.errors(), o.errors(), rtol=EPS_TOL)
    e0, e0o = rec.eps0(pscan["obj"]), o.eps0(pscan["obj"])
    assert abs(e0 - e0o) <= EPS_TOL * e0o


def test_periodic_fixed_point_and_blind_step(pscan, oracle):
    cfg, rec = pscan["cfg"], pscan["rec"]
    z0 = synth.exit_waves(cfg, pscan["obj"], pscan["wt"], pscan["pos"]).astype(np.complex64)
    rec.set_probe(pscan["wt"])
    rec.set_frames(z0)
    rec.iterate(5, cfg.beta)
    assert rel(rec.get_frames().cpu().numpy(), z0) < 5e-6           # noise-free data: the solution is a fixed point (P4)
    assert rec.eps0(pscan["obj"]) < 1e-5
    # one blind iteration from a perturbed probe (Eq. 10 with wrapped object indices)
    w1 = (pscan["wt"] * (1 + 0.2 * _rc(pscan["wt"].shape, 85))).astype(np.complex64)
    rec.set_probe(w1)
    rec.set_probe_refine(1)
    rec.set_frames(z0)
    o = oracle.Oracle(cfg.m, pscan["pos"], pscan["shape"], pscan["I"], w1, refine_every=1)
    o.set_frames(z0)
    rec.iterate(1, cfg.beta)
    o.iterate(1, cfg.beta)
    assert rel(rec.get_frames().cpu().numpy(), o.z) < OP_TOL
    assert rel(rec.get_probe().cpu().numpy(), o.w) < 3e-5
    rec.set_probe_refine(0)
    rec.set_probe(pscan["wt"])


# ---- boundary behaviour ---------------------------------------------------------------------------------------------
def test_misaligned_device_pointers_are_refused(scan):
    """The kernels use 128-bit accesses: a caller pointer that is only 8-byte aligned (a complex64 view with an odd
    storage offset) is SHARP_EINVAL, not a misaligned-address fault."""
    import torch
    cfg, rec = scan["cfg"], scan["rec"]
    m = cfg.m
    buf = torch.zeros(m * m + 1, dtype=torch.complex64, device="cuda")
    odd = buf[1:]
    assert odd.data_ptr() % 16 == 8 and odd.is_contiguous()
    with pytest.raises(sharp.SharpError) as e:
        rec.set_probe(odd)
    assert e.value.code == sharp.SHARP_EINVAL
    big = torch.zeros(cfg.K * m * m + 1, dtype=torch.complex64, device="cuda")
    with pytest.raises(sharp.SharpError) as e:
        rec.op_pa(big[1:])
    assert e.value.code == sharp.SHARP_EINVAL
    rec.set_probe(scan["wt"])                      # the plan is still usable
    assert np.isfinite(rec.get_probe().cpu().numpy()).all()


def test_deferred_and_flushed_blind_paths_agree(scan, oracle):
    """After an illumination update the library defers Q*Q, the cross term and the re-gathered object estimate to the next
    iteration's overlap pass (OV_BLIND); any reader (errors, get_object, eps0) flushes them at once instead.  Both orders
    must give the oracle's state."""
    cfg, rec = scan["cfg"], scan["rec"]
    m = cfg.m
    z0 = (synth.exit_waves(cfg, scan["obj"], scan["w0"], scan["pos"]) * (1 + 0.2 * _rc((cfg.K, m, m), 91))).astype(np.complex64)
    o = oracle.Oracle(m, scan["pos"], scan["shape"], scan["I"], scan["w0"], refine_every=1)
    o.set_frames(z0)
    o.iterate(3, cfg.beta)
    runs = []
    for flush in (False, True):
        rec.set_probe(scan["w0"])
        rec.set_probe_refine(1)
        rec.set_frames(z0)
        if flush:
            for _ in range(3):
                rec.iterate(1, cfg.beta)
                rec.errors(); rec.get_object()             # forces OV_DEN + OV_REGATHER right after every update
        else:
            rec.iterate(3, cfg.beta)                        # two OV_BLIND passes inside
        runs.append((rec.get_frames().cpu().numpy(), rec.get_probe().cpu().numpy(), rec.errors(), rec.get_object().cpu().numpy()))
    for z, w, eps, psi in runs:
        assert rel(z, o.z) < 5e-5 and rel(w, o.w) < 5e-5
        assert np.allclose(eps, o.errors(), rtol=EPS_TOL)
    assert rel(runs[0][0], runs[1][0]) < 2e-5
    den = oracle.overlap_den(o.w, scan["pos"], scan["shape"])
    lit = den >= 1e-3 * den.max()
    assert rel(runs[0][3][lit], runs[1][3][lit]) < 2e-5 and rel(runs[0][3][lit], o.object()[lit]) < 5e-5
    rec.set_probe_refine(0)
    rec.set_probe(scan["wt"])
