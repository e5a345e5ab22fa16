"""B200-native SHARP projection loop (arXiv 1602.01448): ctypes binding over the C-ABI library
`libsharp_b200.so` (include/sharp_b200.h).

The binding only marshals arguments: every step of the method runs in the library's CUDA kernels.  PyTorch is
used for device memory and streams, nothing else.  The library is loaded on first use and the load fails loudly
if it has not been built (`python -c "import __graft_entry__ as g; g.build()"`); there is no CPU fallback.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsharp_b200.so")
HEADER_PATH = os.path.join(os.path.dirname(_HERE), "include", "sharp_b200.h")

SHARP_OK, SHARP_EINVAL, SHARP_ESTATE, SHARP_ENOMEM, SHARP_ECUDA = 0, -1, -2, -3, -4
TILE = 32

_vp, _i, _f, _sz, _ll = C.c_void_p, C.c_int, C.c_float, C.c_size_t, C.c_longlong
_SIGNATURES = {
    "sharp_plan": (_i, [C.POINTER(_vp), _i, _i, _vp, _i, _i]),
    "sharp_plan_periodic": (_i, [C.POINTER(_vp), _i, _i, _vp, _i, _i]),
    "sharp_destroy": (None, [_vp]),
    "sharp_last_error": (C.c_char_p, [_vp]),
    "sharp_workspace_bytes": (_sz, [_vp]),
    "sharp_bind": (_i, [_vp, _vp, _sz, _vp]),
    "sharp_set_intensities": (_i, [_vp, _vp]),
    "sharp_set_probe": (_i, [_vp, _vp]),
    "sharp_set_object": (_i, [_vp, _vp]),
    "sharp_set_frames": (_i, [_vp, _vp]),
    "sharp_set_probe_refine": (_i, [_vp, _i]),
    "sharp_set_frame_slots": (_i, [_vp, _i]),
    "sharp_iterate": (_i, [_vp, _i, _f]),
    "sharp_get_object": (_i, [_vp, _vp]),
    "sharp_get_probe": (_i, [_vp, _vp]),
    "sharp_get_frames": (_i, [_vp, _vp]),
    "sharp_get_amplitudes": (_i, [_vp, _vp]),
    "sharp_errors": (_i, [_vp, C.POINTER(_f)]),
    "sharp_sync": (_i, [_vp]),
    "sharp_launch_count": (_ll, [_vp]),
    "sharp_profile": (_i, [_vp, _i]),
    "sharp_profile_read": (_i, [_vp, C.POINTER(C.c_double), C.POINTER(_ll)]),
    "sharp_tile_grid": (_i, [_vp, C.POINTER(_i), C.POINTER(_i)]),
    "sharp_tile_lists": (_i, [_vp, C.POINTER(_vp), C.POINTER(_vp)]),
    "sharp_cover_counts": (_i, [_vp, _vp]),
    "sharp_frame_index": (_i, [_vp, _vp]),
    "sharp_op_split": (_i, [_vp, _vp, _vp]),
    "sharp_op_overlap": (_i, [_vp, _vp, _vp]),
    "sharp_op_pa": (_i, [_vp, _vp, _vp]),
    "sharp_op_fft2": (_i, [_vp, _vp, _vp, _i]),
    "sharp_op_probe": (_i, [_vp, _vp, _vp, _vp]),
    "sharp_eps0": (_i, [_vp, _vp, _vp, C.POINTER(_f)]),
    "sharp_init_probe": (_i, [_vp]),
    "sharp_init_object_random": (_i, [_vp, C.c_ulonglong]),
    "sharp_op_random_object": (_i, [_vp, C.c_ulonglong, _vp]),
    "sharp_set_sharded": (_i, [_vp, _vp, _vp, _ll]),
    "sharp_set_probe_constraint": (_i, [_vp, _i, _vp]),
    "sharp_set_probe_recentre": (_i, [_vp, _i]),
    "sharp_get_probe_shift": (_i, [_vp, C.POINTER(C.c_int32), C.POINTER(C.c_int32)]),
    "sharp_op_probe_constrain": (_i, [_vp, _vp, _vp]),
    "sharp_fft2_noalloc": (_i, [_vp, _vp, _i, _i, _i, _vp]),
    "sharp_reconstruct_host": (_i, [_vp, _vp, _vp, _i, _f, _vp, _vp, C.POINTER(_f)]),
}

_lib = None


class SharpError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"sharp_b200 error {code}: {text}")
        self.code = code


def load_library():
    """dlopen libsharp_b200.so and bind every symbol include/sharp_b200.h declares.  Raises if the library is
    missing or a symbol is not exported (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} has not been built; run `python -c 'import __graft_entry__ as g; g.build()'`")
        lib = C.CDLL(LIB_PATH)
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(lib, name)          # AttributeError if the symbol is missing
            fn.restype, fn.argtypes = res, args
        _lib = lib
    return _lib


def exported_symbols():
    return sorted(_SIGNATURES)


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else C.c_void_p(None)


NOALLOC_MAX_FRAMES = 4096


def fft2_noalloc(f, out, sign=-1, stream=None):
    """sharp_fft2_noalloc: out <- F f (sign -1) / F* f (sign +1) for K frames of 256 x 256 complex64, with the kernel's
    scratch in a static device array of the library (no plan, no workspace, no allocation inside the call).  `f` and `out`
    are contiguous CUDA complex64 tensors of shape (K, 256, 256) allocated by the caller; asynchronous on `stream`
    (default: torch's current stream).  Calls that overlap on the GPU share the scratch and race."""
    import torch
    lib = load_library()
    assert f.is_cuda and out.is_cuda and f.dtype == out.dtype == torch.complex64 and f.is_contiguous() and out.is_contiguous()
    assert f.shape == out.shape and f.dim() == 3
    st = stream if stream is not None else torch.cuda.current_stream(f.device)
    rc = lib.sharp_fft2_noalloc(_ptr(f), _ptr(out), int(f.shape[-1]), int(f.shape[0]), int(sign), C.c_void_p(st.cuda_stream))
    if rc != SHARP_OK:
        raise SharpError(rc, lib.sharp_last_error(None).decode())
    return out


class Reconstruction:
    """One plan bound to one torch device/stream.  Methods have the names of the C calls without the prefix.
    Array arguments may be numpy arrays or torch tensors; they are moved to the device as float32 / complex64."""

    def __init__(self, m, positions, obj_shape, device="cuda:0", stream=None, periodic=False):
        import torch
        self._torch = torch
        self.lib = load_library()
        self.m = int(m)
        pos = np.ascontiguousarray(positions, dtype=np.int32)
        if pos.ndim != 2 or pos.shape[1] != 2:
            raise ValueError("positions must be (K, 2) int32 (row, col)")
        self.K = int(pos.shape[0])
        self.shape = (int(obj_shape[0]), int(obj_shape[1]))
        self._plan = C.c_void_p(None)
        self.periodic = bool(periodic)
        plan_fn = self.lib.sharp_plan_periodic if self.periodic else self.lib.sharp_plan
        rc = plan_fn(C.byref(self._plan), self.m, self.K, pos.ctypes.data_as(C.c_void_p), *self.shape)
        if rc != SHARP_OK:
            raise SharpError(rc, self.lib.sharp_last_error(None).decode())
        self.device = torch.device(device) if device is not None else None
        self._ws = None
        if self.device is not None:
            if not torch.cuda.is_available():
                raise SharpError(SHARP_ECUDA, "no CUDA device: this library has no CPU path")
            nbytes = int(self.lib.sharp_workspace_bytes(self._plan))
            with torch.cuda.device(self.device):
                self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
                self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
                off = (-self._ws.data_ptr()) % 256
                self._check(self.lib.sharp_bind(self._plan, C.c_void_p(self._ws.data_ptr() + off), nbytes,
                                                C.c_void_p(self._stream.cuda_stream)))

    # -- plumbing ----------------------------------------------------------------------------------------------
    def _check(self, rc):
        if rc != SHARP_OK:
            raise SharpError(rc, self.lib.sharp_last_error(self._plan).decode())

    def _dev(self, x, dtype):
        torch = self._torch
        if x is None:
            return None
        if not torch.is_tensor(x):
            x = torch.from_numpy(np.ascontiguousarray(x))
        with torch.cuda.stream(self._stream):
            return x.to(device=self.device, dtype=dtype, non_blocking=False).contiguous()

    def _new(self, shape, dtype):
        with self._torch.cuda.stream(self._stream):
            return self._torch.empty(shape, dtype=dtype, device=self.device)

    def close(self):
        if getattr(self, "_plan", None) is not None and self._plan.value:
            if self._ws is not None:
                self._torch.cuda.synchronize(self.device)
            self.lib.sharp_destroy(self._plan)
            self._plan = C.c_void_p(None)
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the C calls ---------------------------------------------------------------------------------------------
    def workspace_bytes(self):
        return int(self.lib.sharp_workspace_bytes(self._plan))

    def set_intensities(self, I):
        t = self._dev(I, self._torch.float32)
        assert t.numel() == self.K * self.m * self.m
        self._check(self.lib.sharp_set_intensities(self._plan, _ptr(t)))
        self._keep_I = t    # alive until the stream work is done

    def set_probe(self, w):
        t = self._dev(w, self._torch.complex64)
        assert t.numel() == self.m * self.m
        self._check(self.lib.sharp_set_probe(self._plan, _ptr(t)))
        self._keep_w = t

    def set_object(self, psi=None):
        t = self._dev(psi, self._torch.complex64)
        assert t is None or t.numel() == self.shape[0] * self.shape[1]
        self._check(self.lib.sharp_set_object(self._plan, _ptr(t)))
        self._keep_psi = t

    def set_frames(self, z):
        t = self._dev(z, self._torch.complex64)
        assert t.numel() == self.K * self.m * self.m
        self._check(self.lib.sharp_set_frames(self._plan, _ptr(t)))
        self._keep_z = t

    def set_probe_refine(self, every):
        self._check(self.lib.sharp_set_probe_refine(self._plan, int(every)))

    def set_frame_slots(self, slots):
        self._check(self.lib.sharp_set_frame_slots(self._plan, int(slots)))

    def iterate(self, n, beta):
        self._check(self.lib.sharp_iterate(self._plan, int(n), float(beta)))

    def get_object(self):
        out = self._new(self.shape, self._torch.complex64)
        self._check(self.lib.sharp_get_object(self._plan, _ptr(out)))
        return out

    def get_probe(self):
        out = self._new((self.m, self.m), self._torch.complex64)
        self._check(self.lib.sharp_get_probe(self._plan, _ptr(out)))
        return out

    def get_frames(self):
        out = self._new((self.K, self.m, self.m), self._torch.complex64)
        self._check(self.lib.sharp_get_frames(self._plan, _ptr(out)))
        return out

    def get_amplitudes(self):
        out = self._new((self.K, self.m, self.m), self._torch.float32)
        self._check(self.lib.sharp_get_amplitudes(self._plan, _ptr(out)))
        return out

    def errors(self):
        out = (C.c_float * 3)()
        self._check(self.lib.sharp_errors(self._plan, out))
        return np.array([out[0], out[1], out[2]], dtype=np.float64)

    def sync(self):
        self._check(self.lib.sharp_sync(self._plan))

    def launch_count(self):
        return int(self.lib.sharp_launch_count(self._plan))

    def profile(self, on):
        self._check(self.lib.sharp_profile(self._plan, int(bool(on))))

    def profile_read(self):
        """{class: (summed ms, launches)} for the kernel classes of include/sharp_b200.h (SHARP_PROF_*)."""
        ms, n = (C.c_double * 4)(), (_ll * 4)()
        self._check(self.lib.sharp_profile_read(self._plan, ms, n))
        return {k: (ms[j], int(n[j])) for j, k in enumerate(("frame", "overlap", "probe", "other"))}

    # integer artefacts
    def tile_grid(self):
        a, b = C.c_int(0), C.c_int(0)
        self._check(self.lib.sharp_tile_grid(self._plan, C.byref(a), C.byref(b)))
        return a.value, b.value

    def tile_lists(self):
        tr, tc = self.tile_grid()
        p, f = C.c_void_p(None), C.c_void_p(None)
        self._check(self.lib.sharp_tile_lists(self._plan, C.byref(p), C.byref(f)))
        ptr = np.ctypeslib.as_array(C.cast(p, C.POINTER(C.c_int32)), shape=(tr * tc + 1,)).copy()
        n = int(ptr[-1])
        frames = np.ctypeslib.as_array(C.cast(f, C.POINTER(C.c_int32)), shape=(n,)).copy() if n else np.zeros(0, np.int32)
        return ptr, frames

    def cover_counts(self):
        out = np.empty(self.shape, dtype=np.int32)
        self._check(self.lib.sharp_cover_counts(self._plan, out.ctypes.data_as(C.c_void_p)))
        return out

    def frame_index(self):
        out = self._new((self.K, self.m, self.m), self._torch.int64)
        self._check(self.lib.sharp_frame_index(self._plan, _ptr(out)))
        return out

    # single operators (test hooks)
    def op_split(self, psi):
        t = self._dev(psi, self._torch.complex64)
        out = self._new((self.K, self.m, self.m), self._torch.complex64)
        self._check(self.lib.sharp_op_split(self._plan, _ptr(t), _ptr(out)))
        return out

    def op_overlap(self, f):
        t = self._dev(f, self._torch.complex64)
        out = self._new(self.shape, self._torch.complex64)
        self._check(self.lib.sharp_op_overlap(self._plan, _ptr(t), _ptr(out)))
        return out

    def op_pa(self, f):
        t = self._dev(f, self._torch.complex64)
        out = self._new((self.K, self.m, self.m), self._torch.complex64)
        self._check(self.lib.sharp_op_pa(self._plan, _ptr(t), _ptr(out)))
        return out

    def op_fft2(self, f, sign=-1):
        t = self._dev(f, self._torch.complex64)
        out = self._new((self.K, self.m, self.m), self._torch.complex64)
        self._check(self.lib.sharp_op_fft2(self._plan, _ptr(t), _ptr(out), int(sign)))
        return out

    def op_probe(self, psi, z):
        tp = self._dev(psi, self._torch.complex64)
        tz = self._dev(z, self._torch.complex64)
        out = self._new((self.m, self.m), self._torch.complex64)
        self._check(self.lib.sharp_op_probe(self._plan, _ptr(tp), _ptr(tz), _ptr(out)))
        return out

    # known-solution error, default initialisations, illumination constraints
    def eps0(self, psi0, w0=None):
        tp = self._dev(psi0, self._torch.complex64)
        tw = self._dev(w0, self._torch.complex64)
        assert tp.numel() == self.shape[0] * self.shape[1] and (tw is None or tw.numel() == self.m * self.m)
        out = _f(0.0)
        self._check(self.lib.sharp_eps0(self._plan, _ptr(tp), _ptr(tw), C.byref(out)))
        return float(out.value)

    def init_probe(self):
        self._check(self.lib.sharp_init_probe(self._plan))

    def init_object_random(self, seed):
        self._check(self.lib.sharp_init_object_random(self._plan, C.c_ulonglong(int(seed))))

    def op_random_object(self, seed):
        out = self._new(self.shape, self._torch.complex64)
        self._check(self.lib.sharp_op_random_object(self._plan, C.c_ulonglong(int(seed)), _ptr(out)))
        return out

    def set_sharded(self, allreduce, K_total):
        """This plan holds one rank's frames of a scan of K_total frames; allreduce(t) sums the torch tensor t in place
        over all ranks on the current stream (e.g. lambda t: torch.distributed.all_reduce(t)).  Call before
        set_intensities / set_probe."""
        from .sharding import make_allreduce_callback
        self._ar_fn = make_allreduce_callback(self._ws, allreduce, self._stream) if allreduce is not None else None
        fn = C.cast(self._ar_fn, _vp) if self._ar_fn is not None else _vp(None)
        self._check(self.lib.sharp_set_sharded(self._plan, fn, None, int(K_total)))

    def set_probe_constraint(self, kind, con=None):
        kind = {"none": 0, "mask": 1, "amplitude": 2}.get(kind, kind)
        t = self._dev(con, self._torch.float32)
        assert t is None or t.numel() == self.m * self.m
        self._check(self.lib.sharp_set_probe_constraint(self._plan, int(kind), _ptr(t)))

    def set_probe_recentre(self, on):
        self._check(self.lib.sharp_set_probe_recentre(self._plan, int(bool(on))))

    def get_probe_shift(self):
        last, total = (C.c_int32 * 2)(), (C.c_int32 * 2)()
        self._check(self.lib.sharp_get_probe_shift(self._plan, last, total))
        return (int(last[0]), int(last[1])), (int(total[0]), int(total[1]))

    def op_probe_constrain(self, w):
        t = self._dev(w, self._torch.complex64)
        out = self._new((self.m, self.m), self._torch.complex64)
        self._check(self.lib.sharp_op_probe_constrain(self._plan, _ptr(t), _ptr(out)))
        return out

    def reconstruct_host(self, I_host, w_host, n, beta, want_eps=True):
        """HOST buffers in, HOST buffers out (torch CPU tensors, ideally pinned).  Returns (psi, w, eps)."""
        torch = self._torch
        assert I_host.dtype == torch.float32 and I_host.is_contiguous() and not I_host.is_cuda
        assert w_host.dtype == torch.complex64 and w_host.is_contiguous() and not w_host.is_cuda
        if getattr(self, "_host_out", None) is None:
            self._host_out = (torch.empty(self.shape, dtype=torch.complex64).pin_memory(),
                              torch.empty((self.m, self.m), dtype=torch.complex64).pin_memory())
        psi, w = self._host_out
        eps = (C.c_float * 3)()
        self._check(self.lib.sharp_reconstruct_host(self._plan, _ptr(I_host), _ptr(w_host), int(n), float(beta),
                                                    _ptr(psi), _ptr(w), eps if want_eps else None))
        return psi, w, np.array([eps[0], eps[1], eps[2]], dtype=np.float64)
