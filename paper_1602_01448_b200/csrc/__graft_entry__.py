"""Driver entry points: build() compiles every native piece (the sm_100a C-ABI library and the C oracle);
smoke() runs one small invocation of the hot path on cuda:0 and checks it against the oracle."""
from __future__ import annotations

import os
import sys

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def build() -> None:
    from paper_1602_01448_b200 import build as _b
    _b.build()
    import paper_1602_01448_b200 as pkg
    pkg.load_library()                      # dlopen + symbol check; needs no GPU
    from oracle import sharp_oracle         # building the checker is not using it
    sharp_oracle.build()


def smoke() -> None:
    import numpy as np
    import torch
    import paper_1602_01448_b200 as sharp
    from paper_1602_01448_b200 import synth
    from oracle import sharp_oracle as orc

    assert torch.cuda.is_available(), "smoke() needs a CUDA device"
    cfg = synth.reduced(synth.config(1), 5)          # 25 frames of 64x64, the tiny-scan recipe
    pos, shape, I, w0, obj, wt = synth.make(cfg)
    rec = sharp.Reconstruction(cfg.m, pos, shape, device="cuda:0")
    rec.set_intensities(I)
    rec.set_probe(w0)
    rec.set_object(None)
    rec.iterate(3, cfg.beta)
    z = rec.get_frames().cpu().numpy()
    eps = rec.errors()
    o = orc.Oracle(cfg.m, pos, shape, I, w0)
    o.iterate(3, cfg.beta)
    rel = np.linalg.norm(z - o.z) / np.linalg.norm(o.z)
    eo = o.errors()
    print(f"smoke: frames rel-L2 vs oracle after 3 RAAR iterations = {rel:.3e}; eps gpu={eps} oracle={eo}")
    assert rel < 1e-4, rel
    assert np.allclose(eps, eo, rtol=1e-3), (eps, eo)


if __name__ == "__main__":
    build()
    if len(sys.argv) > 1 and sys.argv[1] == "smoke":
        smoke()
