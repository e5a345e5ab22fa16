"""Host-side plumbing of the sharded reconstruction (include/sharp_b200.h, sharp_set_sharded; Fig. 2):
the partition of the frames over the ranks by spatial region and the adapter that turns a torch collective into the
C callback the library calls.  No step of the method is computed here."""
from __future__ import annotations

import ctypes as C

import numpy as np

ALLREDUCE_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_void_p, C.c_size_t, C.c_int)


def rank_grid(world: int):
    """world = pr x pc with pr <= pc as square as possible (Fig. 2 shows 2 x 2 for 4 GPUs)."""
    pr = int(np.floor(np.sqrt(world)))
    while world % pr:
        pr -= 1
    return pr, world // pr


def partition_by_region(positions, world: int):
    """Frame indices of every rank: the scan is cut into pr row bands of equal frame count (by row position) and each
    band into pc column cells of equal frame count ("we expect a very even division").  Every frame
    belongs to exactly one rank; the order inside a rank is ascending frame index.  Returns a list of int64 arrays."""
    pos = np.asarray(positions)
    K = len(pos)
    pr, pc = rank_grid(world)
    order_r = np.lexsort((np.arange(K), pos[:, 1], pos[:, 0]))          # by row, then column, then index
    parts = []
    for band in np.array_split(order_r, pr):
        by_col = band[np.lexsort((band, pos[band, 0], pos[band, 1]))]
        for cell in np.array_split(by_col, pc):
            parts.append(np.sort(cell).astype(np.int64))
    return parts


def make_allreduce_callback(workspace, allreduce, stream=None):
    """C callback for sharp_set_sharded.  `workspace` is the torch uint8 tensor that holds the plan's workspace (device,
    or CPU in the host-side tests); `allreduce(t)` must sum the torch tensor t in place over all ranks (for example
    `lambda t: torch.distributed.all_reduce(t)`); `stream` is the torch CUDA stream the plan is bound to: the collective
    is enqueued under it, so it is ordered with the library's kernels."""
    import torch

    base = workspace.data_ptr()
    nbytes = workspace.numel()

    def view(ptr, count, is_double):
        off = int(ptr) - base
        size = int(count) * (8 if is_double else 4)
        if off < 0 or off + size > nbytes:
            raise ValueError("all-reduce request outside the plan's workspace")
        return workspace[off:off + size].view(torch.float64 if is_double else torch.float32)

    def cb(user, ptr, count, is_double):
        try:
            t = view(ptr, count, is_double)
            if stream is not None:
                with torch.cuda.stream(stream):
                    allreduce(t)
            else:
                allreduce(t)
            return 0
        except Exception as e:                      # never let an exception cross the C ABI
            cb.last_error = e
            return 1

    cb.last_error = None
    fn = ALLREDUCE_FN(cb)
    fn._py = cb                                     # keeps the closure (and its error slot) reachable
    return fn
