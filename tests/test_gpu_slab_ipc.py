"""Slab decomposition, peer mode ACROSS PROCESSES (fcg_slab_ipc_export / fcg_slab_ipc_open): two processes,
one rank each, exchange the CUDA IPC handles of their workspaces and then run one solve in which the row pass of each stores its
lines straight into the other's exchange buffer and the column pass scatters straight into the other's T2.

This pool has one GPU per run, so both processes use cuda:0 (IPC between processes on one device is the same API as between
devices; the NVLink path itself is not exercised).  No kernel waits on another: every pass is its own launch and the barriers
between the passes are host-side collectives (gloo all-reduce on a device token, which is ordered after the rank's preceding
kernels), so the two processes may time-slice the GPU in any order."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out, L):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    from oracle import api as orc
    from paper_1305_3625_b200 import inputs, slab
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    torch.cuda.set_device(0)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = inputs.config(1, np.float64, L=L)
    to = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    comm = slab.DistComm()
    r = slab.SlabRank(L, torch.float64, world, rank, to(w.s))
    slab.connect_peers_dist(r, comm)
    k, f, u = [to(w.k[r.rows])], [to(w.f[r.rows])], [to(w.u0[r.rows])]
    it, rr, st = slab.slab_solve([r], comm, k, f, u, w.tol, w.maxit)
    ref = orc.cg(w.s, w.k, w.f, w.u0, w.tol, w.maxit)
    mine = u[0].cpu().numpy()
    err = float(np.linalg.norm(mine - ref["u"][r.rows]) / np.linalg.norm(ref["u"][r.rows]))
    # a second solve on the same mappings (warm start from the solution: zero iterations)
    it2, _, st2 = slab.slab_solve([r], comm, k, f, u, 10 * w.tol, w.maxit)
    out[rank] = (it, rr, st, ref["iters"], err, it2, st2)
    dist.barrier()
    r.close()
    dist.destroy_process_group()


@pytest.mark.timeout(600)
def test_slab_peer_mode_two_processes_ipc():
    assert torch.cuda.is_available()
    world, L = 2, 256
    mgr = mp.get_context("spawn").Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), out, L), nprocs=world, join=True)
    assert out[0][:3] == out[1][:3]                               # count, residual, status identical on both ranks
    for rank in range(world):
        it, rr, st, it_or, err, it2, st2 = out[rank]
        assert st == 0 and abs(it - it_or) <= 2 and rr <= 1e-10
        assert err <= 1e-9, (rank, err)
        assert (it2, st2) == (0, 0)
