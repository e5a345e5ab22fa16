"""Sharded reconstruction: frames partitioned over ranks by region, every
sum over frames completed by an all-reduce.

CPU part (`-m "not gpu"`): the partition, and on a world-size-2 gloo group (a) the callback adapter that the binding
hands to sharp_set_sharded really sums a workspace slice over the ranks, (b) the exchange list is the right one: the
oracle's operators evaluated per rank on its frames, with exactly the quantities the library all-reduces (||a||^2, Q*Q,
the object numerator, the Eq. 10 sums, the residual sums) summed over ranks, reproduce the unsharded oracle.

GPU part: two ranks as two host threads on one GPU (own plans, own streams; the all-reduce is emulated on the host side
with a barrier, so no kernel ever waits for another), compared with the oracle on the whole scan."""
import os
import socket
import threading

import numpy as np
import pytest

import synth
from paper_1602_01448_b200.sharding import ALLREDUCE_FN, make_allreduce_callback, partition_by_region, rank_grid


def rel(a, b):
    a = np.asarray(a); b = np.asarray(b)
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))


# ---- partition ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("world", [1, 2, 3, 4, 6, 8])
def test_partition_is_a_balanced_partition_by_region(world):
    for n in (2, 5):
        pos = synth.positions(synth.reduced(synth.config(n), 12 if n == 2 else 150))
        parts = partition_by_region(pos, world)
        assert len(parts) == world and rank_grid(world)[0] * rank_grid(world)[1] == world
        allidx = np.concatenate(parts)
        assert np.array_equal(np.sort(allidx), np.arange(len(pos)))                  # every frame exactly once
        sizes = [len(p) for p in parts]
        assert max(sizes) - min(sizes) <= 2                                            # "very even division"
        assert all(np.all(np.diff(p) > 0) for p in parts)                              # ascending inside a rank
        if world == 2:                                                                  # regions: a left and a right half
            assert pos[parts[0], 1].max() <= pos[parts[1], 1].min() + 0


# ---- world-size-2 gloo ----------------------------------------------------------------------------------------------
def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _gloo_worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    from oracle import sharp_oracle as orc
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # (a) the callback adapter on a CPU "workspace"
        ws = torch.zeros(4096, dtype=torch.uint8)
        f32 = ws[256:256 + 40].view(torch.float32); f32[:] = torch.arange(10, dtype=torch.float32) * (rank + 1)
        f64 = ws[512:512 + 24].view(torch.float64); f64[:] = torch.tensor([1.0, 2.0, 3.0], dtype=torch.float64) + rank
        fn = make_allreduce_callback(ws, lambda t: dist.all_reduce(t))
        assert fn(None, ws.data_ptr() + 256, 10, 0) == 0 and fn(None, ws.data_ptr() + 512, 3, 1) == 0
        assert torch.equal(f32, torch.arange(10, dtype=torch.float32) * 3)
        assert torch.equal(f64, torch.tensor([3.0, 5.0, 7.0], dtype=torch.float64))
        assert fn(None, ws.data_ptr() + 4090, 10, 0) == 1                              # outside the workspace: refused

        # (b) the exchange list, with the oracle's operators per rank
        cfg = synth.reduced(synth.config(3), 4)
        pos, shape, I, w0, obj, wt = synth.make(cfg)
        mine = partition_by_region(pos, world)[rank]
        lp, lI = pos[mine], I[mine]
        allsum = lambda x: (dist.all_reduce(t := torch.from_numpy(np.ascontiguousarray(x))), t.numpy())[1]
        a, A2_loc, _, _ = orc.amplitudes(lI)
        A2 = float(allsum(np.array([A2_loc]))[0])                                      # ||a||^2 over the whole scan
        thr = orc.TAU * np.sqrt(A2 / (cfg.K * cfg.m * cfg.m))
        w = w0.astype(np.complex128)
        den = allsum(orc.overlap_den(w, lp, shape))                                    # Q*Q
        z = orc.split(np.ones(shape, complex), w, lp)
        L = lambda f: np.where(den > 0, allsum(orc.overlap_num(f, w, lp, shape)) / np.where(den > 0, den, 1), 0)
        beta = cfg.beta
        y = orc.Pa(z, a, thr)
        psi_y, psi_z = L(y), L(z)                                                      # the object numerators, summed
        z1 = beta * orc.split(2 * psi_y - psi_z, w, lp) + (1 - 2 * beta) * y + beta * z
        psi1 = L(z1)
        # Eq. 10 sums over ranks
        r = np.arange(cfg.m)
        T = psi1[lp[:, 0, None, None] + r[None, :, None], lp[:, 1, None, None] + r[None, None, :]]
        pn, pd = allsum((np.conj(T) * z1).sum(0)), allsum((np.abs(T) ** 2).sum(0))
        w1 = np.where(pd > 0, pn / np.where(pd > 0, pd, 1), w)
        # residual sums
        den1 = allsum(orc.overlap_den(w1, lp, shape))
        pq = orc.split(np.where(den1 > 0, allsum(orc.overlap_num(z1, w1, lp, shape)) / np.where(den1 > 0, den1, 1), 0), w1, lp)
        sums = allsum(np.array([np.sum(np.abs(orc.Pa(z1, a, thr) - z1) ** 2), np.sum(np.abs(pq - z1) ** 2), np.sum(np.abs(z1 - z) ** 2)]))
        eps = np.sqrt(sums / A2)
        # the unsharded oracle on the whole scan
        o = orc.Oracle(cfg.m, pos, shape, I, w0, refine_every=1)
        o.iterate(1, beta)
        out[rank] = (rel(z1, o.z[mine]), rel(w1, o.w), float(np.abs(eps / o.errors() - 1).max()))
    finally:
        dist.destroy_process_group()


def test_gloo_world2_callback_and_exchange_list():
    import torch.multiprocessing as mp
    port = _free_port()
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_gloo_worker, args=(2, port, out), nprocs=2, join=True)
    assert sorted(out.keys()) == [0, 1]
    for rank in (0, 1):
        ez, ew, ee = out[rank]
        assert ez < 1e-12 and ew < 1e-12 and ee < 1e-12, out[rank]


# ---- two ranks on one GPU -----------------------------------------------------------------------------------------------
class _HostAllReduce:
    """Sum over `world` host threads sharing one GPU: every thread brings its tensor, the sum is formed in rank order
    (so all ranks get the same bits) and copied back.  All waiting is done by host threads on a barrier after a device
    synchronisation; no kernel waits on another."""

    def __init__(self, world):
        import torch
        self.torch, self.world = torch, world
        self.bar = threading.Barrier(world)
        self.slots = [None] * world
        self.calls = 0

    def reducer(self, rank):
        torch = self.torch

        def allreduce(t):
            torch.cuda.synchronize()
            self.slots[rank] = t
            self.bar.wait()
            total = self.slots[0].clone()
            for j in range(1, self.world):
                total += self.slots[j]
            torch.cuda.synchronize()
            self.bar.wait()
            t.copy_(total)
            torch.cuda.synchronize()
            self.bar.wait()
            if rank == 0:
                self.calls += 1
        return allreduce


@pytest.mark.gpu
@pytest.mark.parametrize("name,cfgno,grid,world", [("m64", 1, 6, 2), ("m128-blind", 3, 5, 2), ("m256", 4, 4, 3), ("m128-4", 2, 6, 4)])
def test_sharded_reconstruction_matches_the_oracle(oracle, name, cfgno, grid, world):
    import torch
    import paper_1602_01448_b200 as sharp
    cfg = synth.reduced(synth.config(cfgno), grid)
    pos, shape, I, w0, obj, wt = synth.make(cfg)
    parts = partition_by_region(pos, world)
    hub = _HostAllReduce(world)
    rng = np.random.default_rng(7)
    z0 = (synth.exit_waves(cfg, obj, w0, pos) * (1 + 0.2 * (rng.standard_normal((cfg.K, cfg.m, cfg.m)) + 0j))).astype(np.complex64)
    results, errors_ = [None] * world, []

    def run(rank):
        try:
            mine = parts[rank]
            stream = torch.cuda.Stream()
            rec = sharp.Reconstruction(cfg.m, pos[mine], shape, stream=stream)
            rec.set_sharded(hub.reducer(rank), cfg.K)
            rec.set_intensities(I[mine])
            rec.set_probe(w0)
            rec.set_probe_refine(cfg.refine_every)
            rec.set_frames(z0[mine])
            obj0 = rec.get_object().cpu().numpy()
            rec.iterate(2, cfg.beta)
            res = dict(z=rec.get_frames().cpu().numpy(), eps=rec.errors(), psi=rec.get_object().cpu().numpy(),
                       w=rec.get_probe().cpu().numpy(), eps0=rec.eps0(obj, wt), obj0=obj0)
            rec.init_probe()
            res["w_init"] = rec.get_probe().cpu().numpy()
            results[rank] = res
            rec.close()
        except BaseException as e:                      # a dead rank would leave the others at the barrier
            errors_.append((rank, e))
            hub.bar.abort()

    threads = [threading.Thread(target=run, args=(r,)) for r in range(world)]
    [t.start() for t in threads]
    [t.join(timeout=300) for t in threads]
    assert not errors_, errors_
    assert hub.calls > 0

    o = oracle.Oracle(cfg.m, pos, shape, I, w0, refine_every=cfg.refine_every)
    o.set_frames(z0)
    den = oracle.overlap_den(w0, pos, shape)
    lit = den >= 1e-3 * den.max()
    psi_start = o.object()
    o.iterate(2, cfg.beta)
    for rank in range(world):
        r = results[rank]
        assert rel(r["obj0"][lit], psi_start[lit]) < 1e-5
        assert rel(r["z"], o.z[parts[rank]]) < 3e-5, (name, rank)
        assert np.allclose(r["eps"], o.errors(), rtol=1e-4), (r["eps"], o.errors())
        assert rel(r["w"], o.w) < 3e-5
        den2 = oracle.overlap_den(o.w, pos, shape)
        lit2 = den2 >= 1e-3 * den2.max()
        assert rel(r["psi"][lit2], o.object()[lit2]) < 3e-5
        e0 = o.eps0(obj, w0=wt)
        assert abs(r["eps0"] - e0) <= 1e-4 * e0
        assert rel(r["w_init"], oracle.default_probe(I)) < 1e-5
        # all ranks hold the same object and illumination, bit for bit
        assert np.array_equal(r["psi"], results[0]["psi"]) and np.array_equal(r["w"], results[0]["w"])


@pytest.mark.gpu
def test_nccl_allreduce_callback_on_the_plan_stream(oracle):
    """The real collective: a one-rank NCCL group (all this box has), `torch.distributed.all_reduce` handed to
    sharp_set_sharded and called back by the library between its kernels on a non-default stream.  With one rank the sum is
    the identity, so the run must reproduce the oracle; what is exercised is the C callback -> torch view of the workspace
    -> NCCL launch ordered on the plan's stream, with no host synchronisation in between."""
    import torch
    import torch.distributed as dist
    import paper_1602_01448_b200 as sharp
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(_free_port()))
    dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
    try:
        cfg = synth.reduced(synth.config(3), 5)
        pos, shape, I, w0, obj, wt = synth.make(cfg)
        rng = np.random.default_rng(11)
        z0 = (synth.exit_waves(cfg, obj, w0, pos) * (1 + 0.2 * (rng.standard_normal((cfg.K, cfg.m, cfg.m)) + 0j))).astype(np.complex64)
        calls = []

        def allreduce(t):
            calls.append((t.dtype, t.numel()))
            dist.all_reduce(t)

        rec = sharp.Reconstruction(cfg.m, pos, shape, stream=torch.cuda.Stream())
        rec.set_sharded(allreduce, cfg.K)
        rec.set_intensities(I)
        rec.set_probe(w0)
        rec.set_probe_refine(1)
        rec.set_frames(z0)
        rec.iterate(3, cfg.beta)
        z, eps, w = rec.get_frames().cpu().numpy(), rec.errors(), rec.get_probe().cpu().numpy()
        rec.close()
        o = oracle.Oracle(cfg.m, pos, shape, I, w0, refine_every=1)
        o.set_frames(z0)
        o.iterate(3, cfg.beta)
        assert rel(z, o.z) < 5e-5 and rel(w, o.w) < 5e-5 and np.allclose(eps, o.errors(), rtol=1e-4)
        nobj = shape[0] * shape[1]
        assert (torch.float64, 1) in calls and (torch.float32, nobj) in calls and (torch.float32, 2 * nobj) in calls
        assert (torch.float32, 3 * cfg.m * cfg.m) in calls and (torch.float64, 3) in calls
    finally:
        dist.destroy_process_group()
