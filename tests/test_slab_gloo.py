"""Slab decomposition without a GPU: the shape algebra that libfcg exports as
pure host arithmetic (fcg_slab_shape_of), and the exchange of paper_1305_3625_b200/slab.py's DistComm between two gloo ranks.

A synthetic global half spectrum T2[column block][row pair][line] whose every byte-line encodes its own coordinates is split by
rows (what the row passes write: S), exchanged with DistComm.all_to_all, viewed the way fcg_slab_cols' 5-D tensor map reads it (R[source][block]
[local row pair] as C[block][source * Al + local row pair]), and must then be exactly the columns the rank owns with ALL row pairs;
the way back (all_to_all) must restore S.  The all-reduce leg is checked with the scalar block's two doubles."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _global_t2(shape0, L):
    """uint8 [column blocks][row pairs][line bytes]: bytes 0-3 of a line = its column block, 4-7 = its row pair (int32 each)."""
    MB, lb = shape0["column_blocks"], shape0["line_bytes"]
    t = np.zeros((MB, L // 2, lb // 4), np.int32)
    t[:, :, 0] = np.arange(MB)[:, None]
    t[:, :, 1] = np.arange(L // 2)[None, :]
    t[:, :, 2] = 7
    return t.view(np.uint8).reshape(MB, L // 2, lb)


def _worker(rank, world, port, out, L):
    sys.path.insert(0, ROOT)
    from paper_1305_3625_b200 import binding, slab
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    sh = binding.fcg_slab_shape_of(L, torch.float64, world, rank)
    Al, MBl, lb = sh["row_pairs_local"], sh["column_blocks_local"], sh["line_bytes"]
    T2 = _global_t2(sh, L)
    S = torch.from_numpy(np.ascontiguousarray(T2[:, rank * Al:(rank + 1) * Al, :]).reshape(-1))     # what the own row passes write
    assert S.numel() == sh["buffer_bytes"] and sh["chunk_bytes"] * world == sh["buffer_bytes"]
    R = torch.zeros_like(S)
    comm = slab.DistComm()
    comm.all_to_all([R], [S])
    Rn = R.numpy().reshape(world, MBl, Al, lb)
    C = np.ascontiguousarray(Rn.transpose(1, 0, 2, 3)).reshape(MBl, world * Al, lb)                 # the column pass's view of R
    ok_fwd = np.array_equal(C, T2[rank * MBl:(rank + 1) * MBl])                                      # my columns, every row pair
    R2 = torch.from_numpy(np.ascontiguousarray(C.reshape(MBl, world, Al, lb).transpose(1, 0, 2, 3)).reshape(-1))   # .. and what it leaves there
    S2 = torch.zeros_like(S)
    comm.all_to_all([S2], [R2])
    ok_back = torch.equal(S2, S)
    x = torch.tensor([1.0 + rank, 10.0 * (rank + 1)], dtype=torch.float64)
    comm.all_reduce([x])
    out[rank] = (ok_fwd, ok_back, x.tolist(), sh["column0"], sh["columns_local"], sh["rows_local"])
    dist.destroy_process_group()


@pytest.mark.timeout(180)
def test_slab_exchange_world2():
    world, L = 2, 256
    mgr = mp.get_context("spawn").Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), out, L), nprocs=world, join=True)
    for rank in range(world):
        ok_fwd, ok_back, x, col0, ncol, nrow = out[rank]
        assert ok_fwd and ok_back
        assert x == [3.0, 30.0]
        assert (col0, ncol, nrow) == (rank * L // 4, L // 4, L // 2)


def test_slab_shape_algebra():
    """fcg_slab_shape_of for every supported split: the pieces tile the half spectrum and the vectors exactly; bad splits refuse."""
    sys.path.insert(0, ROOT)
    from paper_1305_3625_b200 import binding
    for L in (256, 1024, 2048, 8192):
        for dt, w, nb in ((torch.float64, 8, 4), (torch.float32, 4, 8)):
            for G in (1, 2, 4, 8, 16):
                shapes = [binding.fcg_slab_shape_of(L, dt, G, r) for r in range(G)]
                assert all(s["columns_per_line"] == nb and s["line_bytes"] == 128 for s in shapes)
                assert sum(s["rows_local"] for s in shapes) == L and sum(s["columns_local"] for s in shapes) == L // 2
                assert [s["column0"] for s in shapes] == [r * (L // 2 // G) for r in range(G)]
                assert sum(s["buffer_bytes"] for s in shapes) == L * L * w                       # the half spectrum, once
                assert all(s["column_blocks_local"] * nb == s["columns_local"] for s in shapes)
    for bad in ((2048, 3), (256, 64), (2048, 0)):
        with pytest.raises(binding.FcgError):
            binding.fcg_slab_shape_of(bad[0], torch.float64, bad[1], 0)
    with pytest.raises(binding.FcgError):
        binding.fcg_slab_shape_of(128, torch.float64, 2, 0)                                      # no pipelined engine below L = 256


def test_local_comm_matches_definition():
    """LocalComm (logical ranks in one process) performs the same exchange: out[dst][src chunk] = in[src][dst chunk]."""
    sys.path.insert(0, ROOT)
    from paper_1305_3625_b200 import slab
    G, chunk = 4, 6
    ins = [torch.arange(G * chunk, dtype=torch.uint8) + 40 * g for g in range(G)]
    outs = [torch.zeros(G * chunk, dtype=torch.uint8) for _ in range(G)]
    slab.LocalComm().all_to_all(outs, ins)
    for dst in range(G):
        for src in range(G):
            assert torch.equal(outs[dst][src * chunk:(src + 1) * chunk], ins[src][dst * chunk:(dst + 1) * chunk])
    xs = [torch.tensor([1.0 * g, 2.0], dtype=torch.float64) for g in range(G)]
    slab.LocalComm().all_reduce(xs)
    assert all(x.tolist() == [6.0, 8.0] for x in xs)
