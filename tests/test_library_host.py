"""Host-side checks of the C-ABI library that need no GPU: it loads, exports every symbol include/sharp_b200.h
declares, validates arguments, and its integer artefacts (tile lists, cover counts) equal the oracle's
brute-force enumeration bit for bit."""
import ctypes as C
import re

import numpy as np
import pytest

import paper_1602_01448_b200 as sharp
import synth


@pytest.fixture(scope="module")
def lib():
    from paper_1602_01448_b200 import build
    build.build()
    return sharp.load_library()


def test_library_exports_every_declared_symbol(lib):
    text = open(sharp.HEADER_PATH).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    declared = set(re.findall(r"\b(sharp_[a-z0-9_]+)\s*\(", text))
    assert declared, "no declarations parsed"
    assert declared == set(sharp.exported_symbols())
    for name in declared:
        assert hasattr(lib, name), name


def _plan(lib, m, pos, shape):
    pos = np.ascontiguousarray(pos, dtype=np.int32)
    plan = C.c_void_p(None)
    rc = lib.sharp_plan(C.byref(plan), m, len(pos), pos.ctypes.data_as(C.c_void_p), shape[0], shape[1])
    return rc, plan


def test_plan_rejects_bad_arguments(lib):
    ok_pos = [[0, 0], [10, 20]]
    assert _plan(lib, 64, ok_pos, (100, 100))[0] == sharp.SHARP_OK
    assert _plan(lib, 48, ok_pos, (100, 100))[0] == sharp.SHARP_EINVAL            # m not a supported power of two
    assert _plan(lib, 64, [[0, 37]], (100, 100))[0] == sharp.SHARP_EINVAL         # 37 + 64 > 100
    assert _plan(lib, 64, [[-1, 0]], (100, 100))[0] == sharp.SHARP_EINVAL
    assert _plan(lib, 64, ok_pos, (63, 100))[0] == sharp.SHARP_EINVAL
    assert b"position" in lib.sharp_last_error(None) or b"object" in lib.sharp_last_error(None)
    rc, plan = _plan(lib, 64, ok_pos, (100, 100))
    # nothing is bound: every device call must refuse, loudly, instead of falling back to the CPU
    assert lib.sharp_iterate(plan, 1, 0.75) == sharp.SHARP_ESTATE
    assert lib.sharp_set_probe(plan, None) == sharp.SHARP_ESTATE
    assert lib.sharp_workspace_bytes(plan) > 2 * 2 * 64 * 64 * 8
    lib.sharp_destroy(plan)


@pytest.mark.parametrize("case", ["cfg1", "cfg2-small", "cfg5-small", "random"])
def test_tile_lists_and_cover_counts_bit_exact(lib, oracle, case):
    if case == "cfg1":
        cfg = synth.config(1); pos, shape, m = synth.positions(cfg), cfg.shape, cfg.m
    elif case == "cfg2-small":
        cfg = synth.reduced(synth.config(2), 7); pos, shape, m = synth.positions(cfg), cfg.shape, cfg.m
    elif case == "cfg5-small":
        cfg = synth.reduced(synth.config(5), 30); pos, shape, m = synth.positions(cfg), cfg.shape, cfg.m
    else:
        rng = np.random.default_rng(5)
        m, shape = 64, (301, 173)                         # ragged: not multiples of the tile edge
        pos = np.stack([rng.integers(0, shape[0] - m + 1, 57), rng.integers(0, shape[1] - m + 1, 57)], 1).astype(np.int32)
        pos[0] = (0, 0); pos[1] = (shape[0] - m, shape[1] - m)      # extreme corners
    rec = sharp.Reconstruction(m, pos, shape, device=None)
    tr, tc = rec.tile_grid()
    assert (tr, tc) == (-(-shape[0] // sharp.TILE), -(-shape[1] // sharp.TILE))
    ptr, frames = rec.tile_lists()
    optr, oframes = oracle.tile_lists(m, pos, shape, sharp.TILE)
    assert ptr.dtype == optr.dtype == np.int32
    assert np.array_equal(ptr, optr) and np.array_equal(frames, oframes)
    cnt = rec.cover_counts()
    ocnt = oracle.cover_counts(m, pos, shape)
    assert np.array_equal(cnt, ocnt) and int(cnt.sum()) == len(pos) * m * m          # P7
    rec.close()
