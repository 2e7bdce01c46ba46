"""world_size-2 check (gloo, CPU) of the position sharding used by bench.py --gpus N: each rank
takes its rows, computes loss + gradients on them, the sums are all-reduced; the result must equal the
unsharded pass.  The per-rank pass here is the CPU oracle (tests may call it); on GPUs it is ptycho_gradient."""
import os
import socket

import numpy as np
import pytest

from paper_2505_14372_b200 import shard, synth


def test_shard_rows_partition():
    for n, w in [(10, 3), (4096, 8), (7, 7), (5, 8), (1, 2)]:
        parts = [shard.shard_rows(n, r, w) for r in range(w)]
        cat = np.concatenate(parts)
        assert cat.tolist() == list(range(n))
        assert max(p.size for p in parts) - min(p.size for p in parts) <= 1
    bs = [np.array([5, 3, 9, 1, 0], np.int32), np.array([2, 8], np.int32)]
    a, b = shard.shard_batches(bs, 0, 2), shard.shard_batches(bs, 1, 2)
    assert [x.tolist() for x in a] == [[5, 3, 9], [2]] and [x.tolist() for x in b] == [[1, 0], [8]]
    with pytest.raises(ValueError):
        shard.shard_rows(4, 2, 2)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    from oracle import oracle as orc
    from tests._cases import make_case, oracle_problem
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = synth.config(3, n=64, scan=(3, 3), n_modes=2, n_slices=2, obj_n=120, pixel_size=0.2, step_px=3.0)
    case = make_case(cfg, start_scale=0.8)
    pbo = oracle_problem(cfg)
    rows = shard.shard_rows(cfg.n_pos, rank, world)
    o = orc.gradient(pbo, case.obj_start, case.probe, case.positions, case.intensity, batch_idx=rows, want_illum=True)
    gO = torch.from_numpy(o["grad_object"].astype(np.complex128)); gP = torch.from_numpy(o["grad_probe"].astype(np.complex128))
    il = torch.from_numpy(o["illum"].astype(np.float64)); loss = torch.tensor([o["loss"]], dtype=torch.float64)
    shard.allreduce_sums(dist, gO, gP, il, None, loss)
    if rank == 0:
        full = orc.gradient(pbo, case.obj_start, case.probe, case.positions, case.intensity, want_illum=True)
        err = dict(gO=float(np.abs(gO.numpy() - full["grad_object"]).max() / np.abs(full["grad_object"]).max()),
                   gP=float(np.abs(gP.numpy() - full["grad_probe"]).max() / np.abs(full["grad_probe"]).max()),
                   il=float(np.abs(il.numpy() - full["illum"]).max() / np.abs(full["illum"]).max()),
                   loss=float(abs(loss.item() - full["loss"]) / abs(full["loss"])),
                   gX=float(np.abs(o["grad_pos"] - full["grad_pos"][rows]).max() / np.abs(full["grad_pos"]).max()))
        q.put(err)
    dist.barrier()
    dist.destroy_process_group()


def test_sharded_gradient_equals_unsharded_gloo_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    err = q.get(timeout=240)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert max(err.values()) <= 1e-12, err
