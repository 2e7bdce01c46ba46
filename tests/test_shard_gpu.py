"""Position sharding with the CUDA path as the per-rank pass: two processes, both on
cuda:0 (the box has one GPU; the two passes are independent kernels, neither waits on the other), each runs ptycho_gradient
on ITS shard of the rows through the C ABI, the sums of host copies are all-reduced over gloo, and the result is compared
with the unsharded GPU pass and with the oracle.  Per-position outputs stay with the owning rank and must equal the
unsharded ones bit for bit (each depends on its own position only)."""
import os
import socket

import numpy as np
import pytest

from paper_2505_14372_b200 import shard, synth

pytestmark = pytest.mark.gpu


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _case():
    from tests._cases import make_case
    cfg = synth.config(3, scan=(4, 5), n_modes=4, n_slices=4)
    return cfg, make_case(cfg, start_scale=0.8)


def _gpu_pass(cfg, case, rows):
    import torch
    from paper_2505_14372_b200 import ptycho
    from tests._cases import gpu_problem
    pbg = gpu_problem(cfg)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    obj, pr, pos, inten = dev(case.obj_start), dev(case.probe), dev(case.positions), dev(case.intensity)
    b = None if rows is None else dev(np.asarray(rows, np.int32))
    J = cfg.n_pos if rows is None else len(rows)
    gO, gP = torch.empty_like(obj), torch.empty_like(pr)
    gX = torch.empty((J, 2), dtype=torch.float32, device="cuda")
    il = torch.empty(obj.shape, dtype=torch.float32, device="cuda")
    loss = torch.zeros(1, dtype=torch.float64, device="cuda")
    lpp = torch.empty(J, dtype=torch.float32, device="cuda")
    fl = ptycho.WANT_POS_GRAD | ptycho.WANT_ILLUM
    ws = ptycho.make_workspace(pbg, cfg.n_pos, J, fl)
    ptycho.gradient(pbg, obj, pr, pos, inten, b, workspace=ws, grad_object=gO, grad_probe=gP, grad_pos=gX, illum=il, loss=loss, loss_per_pos=lpp)
    assert ptycho.status(ws) == 0
    return gO.cpu(), gP.cpu(), il.cpu(), loss.cpu(), gX.cpu().numpy(), lpp.cpu().numpy()


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.cuda.set_device(0)
    cfg, case = _case()
    rows = shard.shard_rows(cfg.n_pos, rank, world)
    gO, gP, il, loss, gX, lpp = _gpu_pass(cfg, case, rows)
    shard.allreduce_sums(dist, gO, gP, il, None, loss)
    if rank == 0:
        q.put(dict(gO=gO.numpy(), gP=gP.numpy(), il=il.numpy(), loss=loss.item()))
    q.put(dict(rank=rank, rows=rows, gX=gX, lpp=lpp))
    dist.barrier()
    dist.destroy_process_group()


def test_sharded_gpu_gradient_equals_unsharded_world2():
    import torch.multiprocessing as mp
    from oracle import oracle as orc
    from tests._cases import oracle_problem, rel_l2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = [q.get(timeout=300) for _ in range(3)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    sums = next(g for g in got if "gO" in g)
    per_rank = {g["rank"]: g for g in got if "rank" in g}
    cfg, case = _case()
    gO, gP, il, loss, gX, lpp = _gpu_pass(cfg, case, None)
    # sums over ranks against the one-process pass: the same numbers summed in another order (fp32 outputs of two passes
    # added in fp32 by the all-reduce, against one fp64 accumulation rounded once)
    assert rel_l2(sums["gO"], gO.numpy()) <= 1e-6 and rel_l2(sums["gP"], gP.numpy()) <= 1e-6 and rel_l2(sums["il"], il.numpy()) <= 1e-6
    assert abs(sums["loss"] - loss.item()) <= 1e-12 * abs(loss.item())
    for r in range(2):
        rows = per_rank[r]["rows"]
        assert per_rank[r]["gX"].tobytes() == gX[rows].tobytes() and per_rank[r]["lpp"].tobytes() == lpp[rows].tobytes()
    # and against the oracle over all positions
    o = orc.gradient(oracle_problem(cfg), case.obj_start, case.probe, case.positions, case.intensity, want_illum=True)
    assert rel_l2(sums["gO"], o["grad_object"]) <= 1e-4 and rel_l2(sums["gP"], o["grad_probe"]) <= 1e-4
    assert rel_l2(sums["il"], o["illum"]) <= 1e-4 and abs(sums["loss"] - o["loss"]) <= 1e-5 * abs(o["loss"])
