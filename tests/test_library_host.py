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


@pytest.mark.parametrize("case", ["fig3-small", "random-wrap", "corner"])
def test_periodic_tile_lists_and_cover_counts_bit_exact(lib, oracle, case):
    """sharp_plan_periodic (reading G25): lists and counts against the oracle's brute force over wrapped
    pixels, on shapes that are not multiples of the tile edge."""
    if case == "fig3-small":
        cfg = synth.reduced(synth.config(6), 17); pos, shape, m = synth.positions(cfg), cfg.shape, cfg.m     # 170 x 170
    elif case == "random-wrap":
        rng = np.random.default_rng(6)
        m, shape = 64, (131, 97)                           # 97 - 64 = 33 >= TILE - 1
        pos = np.stack([rng.integers(0, shape[0], 41), rng.integers(0, shape[1], 41)], 1).astype(np.int32)
    else:
        m, shape = 64, (95, 200)                           # the smallest legal margin on rows: 95 - 64 = 31
        pos = np.array([[94, 199], [0, 0], [31, 136], [32, 137], [63, 1]], np.int32)
    rec = sharp.Reconstruction(m, pos, shape, device=None, periodic=True)
    ptr, frames = rec.tile_lists()
    optr, oframes = oracle.tile_lists_periodic(m, pos, shape, sharp.TILE)
    assert np.array_equal(ptr, optr) and np.array_equal(frames, oframes)
    cnt = rec.cover_counts()
    assert np.array_equal(cnt, oracle.cover_counts(m, pos, shape)) and int(cnt.sum()) == len(pos) * m * m
    rec.close()


def test_periodic_plan_validation(lib):
    def plan(m, pos, shape):
        pos = np.ascontiguousarray(pos, dtype=np.int32)
        h = C.c_void_p(None)
        rc = lib.sharp_plan_periodic(C.byref(h), m, len(pos), pos.ctypes.data_as(C.c_void_p), shape[0], shape[1])
        if rc == sharp.SHARP_OK:
            lib.sharp_destroy(h)
        return rc
    assert plan(64, [[99, 99]], (100, 100)) == sharp.SHARP_OK          # anywhere in the image
    assert plan(64, [[100, 0]], (100, 100)) == sharp.SHARP_EINVAL       # but inside it
    assert plan(64, [[0, 0]], (94, 100)) == sharp.SHARP_EINVAL          # margin 30 < TILE - 1
    assert plan(64, [[0, 0]], (95, 95)) == sharp.SHARP_OK
