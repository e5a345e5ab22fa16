"""ctypes face of the CPU ORACLE (oracle/sharp_oracle.c) + the reconstruction sequence of PAPER.md:167-194.

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
``--impl reference`` leg may import this.  It imports nothing from paper_1602_01448_b200 and that package
imports nothing from here.

All arithmetic is in oracle/sharp_oracle.c (double precision, one loop nest per formula).  This file only
marshals numpy arrays and strings the steps together in the paper's order:

  step 4  z0 = Q psi0
  step 5  z  <- RAAR(z)                                PAPER.md:174-178  (sign: DESIGN.md reading G1)
  step 6  psi <- Q* z / Q* Q                           PAPER.md:180, Eq. (9)
  step 7  w  <- Eq. (10) every `refine_every` its      PAPER.md:181       (order: reading G10)
          then the Fourier mask or amplitude constraint and the centre-of-mass shift (:191)

Parity unpinned: see the header of sharp_oracle.c.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sharp_oracle.c")
_LIB = os.path.join(_HERE, "libsharp_oracle.so")

TAU = 1e-4  # G4: thr = TAU * a_rms


def build(force: bool = False) -> str:
    """Compile oracle/sharp_oracle.c -> oracle/libsharp_oracle.so (gcc, -O2, no fast-math, OpenMP)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"])
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
    return _lib


def _c(a):  # complex128, C-contiguous
    return np.ascontiguousarray(a, dtype=np.complex128)


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _pos(pos):
    pos = np.ascontiguousarray(pos, dtype=np.int32)
    assert pos.ndim == 2 and pos.shape[1] == 2
    return pos


def n_threads() -> int:
    """Threads the C oracle's OpenMP loops use on this host."""
    return int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))


# ---- O1 ------------------------------------------------------------------------------------------
def dft2_naive(f, sign=-1):
    f = _c(f); m = f.shape[-1]; assert f.shape == (m, m)
    out = np.empty_like(f)
    lib().orc_dft2_naive(C.c_int(m), _p(f), _p(out), C.c_int(sign))
    return out


def fft2(f, sign=-1):
    f = _c(f); m = f.shape[-1]; assert f.shape == (m, m) and (m & (m - 1)) == 0
    out = np.empty_like(f)
    lib().orc_fft2(C.c_int(m), _p(f), _p(out), C.c_int(sign))
    return out


# ---- O2 ------------------------------------------------------------------------------------------
def amplitudes(I):
    """a = sqrt(max(I,0)), A2 = sum a^2, a_rms, thr = TAU*a_rms  (G4, G12, G14)."""
    I = np.ascontiguousarray(I, dtype=np.float32)
    a = np.empty(I.shape, dtype=np.float64)
    A2 = C.c_double(0.0)
    lib().orc_amplitudes(C.c_long(I.size), _p(I), _p(a), C.byref(A2))
    a_rms = float(np.sqrt(A2.value / I.size))
    return a, A2.value, a_rms, TAU * a_rms


# ---- O3 / O4 -------------------------------------------------------------------------------------
def split(psi, w, pos):
    psi = _c(psi); w = _c(w); pos = _pos(pos)
    m = w.shape[0]; K = pos.shape[0]; nr, nc = psi.shape
    z = np.empty((K, m, m), dtype=np.complex128)
    lib().orc_split(C.c_int(m), C.c_int(K), _p(pos), C.c_int(nr), C.c_int(nc), _p(psi), _p(w), _p(z))
    return z


def overlap_num(f, w, pos, shape):
    f = _c(f); w = _c(w); pos = _pos(pos); K, m, _ = f.shape; nr, nc = shape
    num = np.empty((nr, nc), dtype=np.complex128)
    lib().orc_overlap_num(C.c_int(m), C.c_int(K), _p(pos), C.c_int(nr), C.c_int(nc), _p(w), _p(f), _p(num))
    return num


def overlap_den(w, pos, shape):
    w = _c(w); pos = _pos(pos); m = w.shape[0]; K = pos.shape[0]; nr, nc = shape
    den = np.empty((nr, nc), dtype=np.float64)
    lib().orc_overlap_den(C.c_int(m), C.c_int(K), _p(pos), C.c_int(nr), C.c_int(nc), _p(w), _p(den))
    return den


def L(f, w, pos, shape):
    f = _c(f); w = _c(w); pos = _pos(pos); K, m, _ = f.shape; nr, nc = shape
    psi = np.empty((nr, nc), dtype=np.complex128)
    lib().orc_L(C.c_int(m), C.c_int(K), _p(pos), C.c_int(nr), C.c_int(nc), _p(w), _p(f), _p(psi))
    return psi


def PQ(f, w, pos, shape):
    f = _c(f); w = _c(w); pos = _pos(pos); K, m, _ = f.shape; nr, nc = shape
    out = np.empty_like(f)
    lib().orc_PQ(C.c_int(m), C.c_int(K), _p(pos), C.c_int(nr), C.c_int(nc), _p(w), _p(f), _p(out))
    return out


# ---- O5 / O6 -------------------------------------------------------------------------------------
def Pa(z, a, thr, naive=False):
    z = _c(z); a = np.ascontiguousarray(a, dtype=np.float64); K, m, _ = z.shape
    y = np.empty_like(z)
    lib().orc_Pa(C.c_int(m), C.c_int(K), _p(z), _p(a), C.c_double(thr), _p(y), C.c_int(int(naive)))
    return y


def raar(z, w, pos, shape, a, thr, beta, naive=False, return_y=False):
    z = _c(z); w = _c(w); pos = _pos(pos); a = np.ascontiguousarray(a, dtype=np.float64)
    K, m, _ = z.shape; nr, nc = shape
    zn = np.empty_like(z)
    y = np.empty_like(z) if return_y else None
    lib().orc_raar(C.c_int(m), C.c_int(K), _p(pos), C.c_int(nr), C.c_int(nc), _p(w), _p(a), C.c_double(thr),
                   C.c_double(beta), _p(z), _p(zn), _p(y) if return_y else None, C.c_int(int(naive)))
    return (zn, y) if return_y else zn


def raar_one_split(z, w, pos, shape, a, thr, beta, naive=False):
    z = _c(z); w = _c(w); pos = _pos(pos); a = np.ascontiguousarray(a, dtype=np.float64)
    K, m, _ = z.shape; nr, nc = shape
    zn = np.empty_like(z)
    lib().orc_raar_one_split(C.c_int(m), C.c_int(K), _p(pos), C.c_int(nr), C.c_int(nc), _p(w), _p(a),
                             C.c_double(thr), C.c_double(beta), _p(z), _p(zn), C.c_int(int(naive)))
    return zn


# ---- O8 / O9 -------------------------------------------------------------------------------------
def probe_update(psi, z, w, pos):
    psi = _c(psi); z = _c(z); pos = _pos(pos); K, m, _ = z.shape; nr, nc = psi.shape
    wn = _c(w).copy()
    lib().orc_probe_update(C.c_int(m), C.c_int(K), _p(pos), C.c_int(nr), C.c_int(nc), _p(psi), _p(z), _p(wn))
    return wn


def errors(z, zprev, w, pos, shape, a, thr, A2, naive=False):
    z = _c(z); w = _c(w); pos = _pos(pos); a = np.ascontiguousarray(a, dtype=np.float64)
    K, m, _ = z.shape; nr, nc = shape
    zp = _c(zprev) if zprev is not None else None
    out = (C.c_double * 3)()
    lib().orc_errors(C.c_int(m), C.c_int(K), _p(pos), C.c_int(nr), C.c_int(nc), _p(w), _p(a), C.c_double(thr),
                     C.c_double(A2), _p(z), _p(zp) if zp is not None else None, out, C.c_int(int(naive)))
    return np.array([out[0], out[1], out[2]])


# ---- O10 -----------------------------------------------------------------------------------------
def linear_index(m, pos, nc):
    pos = _pos(pos); K = pos.shape[0]
    idx = np.empty((K, m, m), dtype=np.int64)
    lib().orc_linear_index(C.c_int(m), C.c_int(K), _p(pos), C.c_int(nc), _p(idx))
    return idx


def cover_counts(m, pos, shape):
    pos = _pos(pos); K = pos.shape[0]; nr, nc = shape
    cnt = np.empty((nr, nc), dtype=np.int32)
    lib().orc_cover_counts(C.c_int(m), C.c_int(K), _p(pos), C.c_int(nr), C.c_int(nc), _p(cnt))
    return cnt


def tile_lists(m, pos, shape, T):
    pos = _pos(pos); K = pos.shape[0]; nr, nc = shape
    nt = ((nr + T - 1) // T) * ((nc + T - 1) // T)
    ptr = np.empty(nt + 1, dtype=np.int32)
    lib().orc_tile_lists(C.c_int(m), C.c_int(K), _p(pos), C.c_int(nr), C.c_int(nc), C.c_int(T), _p(ptr), None)
    frames = np.empty(int(ptr[-1]), dtype=np.int32)
    lib().orc_tile_lists(C.c_int(m), C.c_int(K), _p(pos), C.c_int(nr), C.c_int(nc), C.c_int(T), _p(ptr), _p(frames))
    return ptr, frames


# ---- the reconstruction sequence ------------------------------------------------------------------
class Oracle:
    """State (z, w, psi) advanced by steps 5-7 of PAPER.md:174-181.  Inputs are the same f32/c64 arrays the
    GPU library receives, widened to double once."""

    def __init__(self, m, pos, shape, intensities, probe, psi0=None, refine_every=0, probe_mask=None,
                 probe_amplitude=None, recentre=False):
        self.m = int(m); self.pos = _pos(pos); self.shape = tuple(int(s) for s in shape)
        self.K = self.pos.shape[0]
        I = np.asarray(intensities, dtype=np.float32).reshape(self.K, self.m, self.m)
        self.a, self.A2, self.a_rms, self.thr = amplitudes(I)
        self.w = _c(np.asarray(probe).reshape(self.m, self.m))
        self.refine_every = int(refine_every)
        self.mask = None if probe_mask is None else np.asarray(probe_mask, dtype=np.float64)    # m_w
        self.aw = None if probe_amplitude is None else np.asarray(probe_amplitude, dtype=np.float64)   # a_w
        self.recentre = bool(recentre)
        self.shifts = []
        psi0 = np.ones(self.shape, np.complex128) if psi0 is None else _c(psi0)   # G8: flat 1+0i
        self.z = split(psi0, self.w, self.pos)                                      # step 4 (G7)
        self.zprev = None                                                           # "z^(0) = 0" for eps_Delta
        self.psi = L(self.z, self.w, self.pos, self.shape)
        self.it = 0

    def set_frames(self, z, zprev=None):
        """Teacher forcing (tests): overwrite the frame state; psi follows by Eq. (9)."""
        self.z = _c(z).reshape(self.K, self.m, self.m).copy()
        self.zprev = None if zprev is None else _c(zprev).reshape(self.z.shape).copy()
        self.psi = L(self.z, self.w, self.pos, self.shape)

    def iterate(self, n, beta):
        for _ in range(int(n)):
            self.it += 1
            znew = raar(self.z, self.w, self.pos, self.shape, self.a, self.thr, beta)      # step 5
            self.zprev, self.z = self.z, znew
            self.psi = L(self.z, self.w, self.pos, self.shape)                              # step 6
            if self.refine_every and self.it % self.refine_every == 0:                      # step 7
                self.w = probe_update(self.psi, self.z, self.w, self.pos)
                if self.mask is not None:                                                   # "If m_w is given ..."
                    self.w = probe_mask(self.w, self.mask)
                elif self.aw is not None:                                                   # "else if a_w is given ..."
                    self.w = probe_amplitude(self.w, self.aw)
                if self.recentre:                                                           # "Now compute center of mass"
                    self.w, d = probe_recentre(self.w)
                    self.shifts.append(d)
        return self

    def object(self):
        """psi = L_w z with the current w (what sharp_get_object returns)."""
        return L(self.z, self.w, self.pos, self.shape)

    def eps0(self, psi0, w0=None):
        """Eq. (14) at the current frames, against the known solution psi0 (and its illumination w0)."""
        return eps0(self.z, psi0, self.w, self.pos, self.shape, w0=w0)

    def errors(self):
        return errors(self.z, self.zprev, self.w, self.pos, self.shape, self.a, self.thr, self.A2)


# ---- O11-O14: eps_0, default initialisations, illumination constraints, re-centring ---------------------------
def eps0(z, psi0, w, pos, shape, w0=None, return_phi=False):
    """Eq. (14): min_phi ||Q*(e^{i phi} z - z0)|| / ||Q* z0||, z0 = Q_{w0} psi0 (w0 = w if None)."""
    z = _c(z); w = _c(w); w0 = w if w0 is None else _c(w0); psi0 = _c(psi0); pos = _pos(pos)
    K, m, _ = z.shape; nr, nc = shape
    phi = C.c_double(0.0)
    f = lib().orc_eps0; f.restype = C.c_double
    e = f(C.c_int(m), C.c_int(K), _p(pos), C.c_int(nr), C.c_int(nc), _p(w), _p(w0), _p(z), _p(psi0), C.byref(phi))
    return (float(e), phi.value) if return_phi else float(e)


def default_probe(I):
    """PAPER.md:171 step 2: w0 = F*(sqrt(mean frame)), moved to the frame centre (reading G21)."""
    I = np.ascontiguousarray(I, dtype=np.float32); K, m, _ = I.shape
    w0 = np.empty((m, m), dtype=np.complex128)
    lib().orc_default_probe(C.c_int(m), C.c_int(K), _p(I), _p(w0))
    return w0


def random_object(shape, seed):
    """PAPER.md:172 step 3: psi0 ~ U[0,1) from the counter-based generator both sides implement (float32, exact)."""
    nr, nc = shape
    re = np.empty((nr, nc), dtype=np.float32)
    lib().orc_random_object(C.c_long(nr * nc), C.c_uint64(seed), _p(re))
    return re.astype(np.complex128)


def probe_mask(w, mask):
    w = _c(w); m = w.shape[0]; mask = np.ascontiguousarray(mask, dtype=np.float64)
    out = np.empty_like(w)
    lib().orc_probe_mask(C.c_int(m), _p(w), _p(mask), _p(out))
    return out


def probe_amplitude(w, aw, thr_w=None):
    w = _c(w); m = w.shape[0]; aw = np.ascontiguousarray(aw, dtype=np.float64)
    if thr_w is None:
        thr_w = TAU * float(np.sqrt(np.mean(aw * aw)))           # reading G24
    out = np.empty_like(w)
    lib().orc_probe_amplitude(C.c_int(m), _p(w), _p(aw), C.c_double(thr_w), _p(out))
    return out


def probe_recentre(w):
    w = _c(w); m = w.shape[0]
    out = np.empty_like(w)
    d = (C.c_int32 * 2)()
    lib().orc_probe_recentre(C.c_int(m), _p(w), _p(out), d)
    return out, (int(d[0]), int(d[1]))


def linear_index_periodic(m, pos, shape):
    pos = _pos(pos); K = pos.shape[0]; nr, nc = shape
    idx = np.empty((K, m, m), dtype=np.int64)
    lib().orc_linear_index_periodic(C.c_int(m), C.c_int(K), _p(pos), C.c_int(nr), C.c_int(nc), _p(idx))
    return idx


def tile_lists_periodic(m, pos, shape, T):
    pos = _pos(pos); K = pos.shape[0]; nr, nc = shape
    nt = ((nr + T - 1) // T) * ((nc + T - 1) // T)
    ptr = np.empty(nt + 1, dtype=np.int32)
    a = (C.c_int(m), C.c_int(K), _p(pos), C.c_int(nr), C.c_int(nc), C.c_int(T))
    lib().orc_tile_lists_periodic(*a, _p(ptr), None)
    frames = np.empty(int(ptr[-1]), dtype=np.int32)
    lib().orc_tile_lists_periodic(*a, _p(ptr), _p(frames))
    return ptr, frames
