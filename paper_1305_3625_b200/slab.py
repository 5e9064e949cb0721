"""Slab-decomposed CG over several ranks: the ORDER of the library's
local passes and of the two collectives between them.  No arithmetic of the method happens here -- every vector update,
transform, dot product and scalar step is a kernel of libfcg (fcg_slab_* in include/fcg.h); this module only sequences them
and moves the exchange buffers between the ranks:

  * DistComm   one process per GPU (torchrun): torch.distributed all_to_all_single / all_reduce over NCCL on the handle's
               stream; with the gloo backend (CPU tests) the all-to-all is done with isend / irecv, which gloo does have;
  * LocalComm  G logical ranks that share one device and one stream (parity tests on the one-GPU pool): the all-to-all is G*G
               device copies, the all-reduce a sum of G four-element tensors.

Per iteration, with the spectral search length (default; DESIGN.md sections 12 and 18):
    rows_fwd | all-to-all S->R | cols_energy (on R, in place) | all-to-all R->S | all-reduce | scalar(4) | rows_inv(2) | all-reduce | scalar(5)
or in the textbook order of Listing 2:
    rows_fwd | all-to-all S->R | cols | all-to-all R->S | rows_inv | all-reduce | scalar(1) | update_r | all-reduce | scalar(2)
(peer mode: the all-to-alls are barriers, the passes store straight into the peers' buffers), with one read-back of the scalar block every `poll_every` iterations: once the device-side stopping decision has been taken
(identically on every rank) the remaining passes of the chunk return at once without touching anything.
"""
from __future__ import annotations

import torch

from . import binding


class LocalComm:
    """Collectives among logical ranks of ONE process: arguments are lists with one tensor per rank."""

    def all_to_all(self, outs, ins):
        G = len(ins)
        chunk = ins[0].numel() // G
        for dst in range(G):
            for src in range(G):
                outs[dst][src * chunk:(src + 1) * chunk].copy_(ins[src][dst * chunk:(dst + 1) * chunk])

    def all_reduce(self, xs):
        total = torch.stack(list(xs)).sum(dim=0)
        for x in xs:
            x.copy_(total)

    def barrier(self, xs):
        pass                                         # one stream: the launches of all logical ranks are already ordered


class DistComm:
    """Collectives among the processes of torch.distributed's default group: lists of length one (this process's tensors)."""

    def __init__(self):
        import torch.distributed as dist
        self.dist = dist
        self.world, self.rank = dist.get_world_size(), dist.get_rank()
        self.native_a2a = dist.get_backend() == "nccl"

    def all_to_all(self, outs, ins):
        out, inp = outs[0], ins[0]
        if self.native_a2a:
            self.dist.all_to_all_single(out, inp)
            return
        chunk = inp.numel() // self.world                 # gloo: no all_to_all; the same exchange from point-to-point calls
        reqs = []
        for peer in range(self.world):
            if peer == self.rank:
                out[peer * chunk:(peer + 1) * chunk].copy_(inp[peer * chunk:(peer + 1) * chunk])
                continue
            reqs.append(self.dist.isend(inp[peer * chunk:(peer + 1) * chunk].contiguous(), peer))
            reqs.append(self.dist.irecv(out[peer * chunk:(peer + 1) * chunk], peer))
        for r in reqs:
            r.wait()

    def all_reduce(self, xs):
        self.dist.all_reduce(xs[0])

    def barrier(self, xs):
        """Stream-ordered barrier between the ranks: a collective on the stream completes on a rank only after every rank has
        reached it in ITS stream, i.e. after that rank's preceding pass (whose peer stores are then visible) has finished."""
        if not hasattr(self, "_tok"):
            self._tok = torch.zeros(1, dtype=torch.float32, device=xs[0].device)
        self.dist.all_reduce(self._tok)


class SlabRank:
    """One rank's handle, its rows of k, f, u, and its exchange buffers."""

    def __init__(self, L: int, dtype, nranks: int, rank: int, s_full: torch.Tensor, device="cuda"):
        self.shape = binding.fcg_slab_shape_of(L, dtype, nranks, rank)
        self.h = binding.Fcg(L, dtype, device=device)
        self.h.fcg_set_spectrum(s_full)
        self.h.fcg_slab_configure(nranks, rank)
        self.send, self.recv = self.h.fcg_slab_buffers()
        self.xch = torch.zeros(4, dtype=torch.float64, device=device)     # this rank's shares of the iteration's sums, all-reduced in place
        self.rows = slice(rank * self.shape["rows_local"], (rank + 1) * self.shape["rows_local"])

    def close(self):
        self.h.close()


def connect_peers_local(ranks):
    """Logical ranks of one process on one device: every handle gets the addresses of all the others' buffers (peer mode: the
    row pass stores, and the column pass scatters, straight into the destination rank's buffer; include/fcg.h)."""
    send = [r.send.data_ptr() for r in ranks]; recv = [r.recv.data_ptr() for r in ranks]
    for r in ranks:
        r.h.fcg_slab_set_peers(send, recv)
        r.peers = True


def connect_peers_dist(rank_obj, comm):
    """One process per GPU: exchange the CUDA IPC blobs of the workspaces (a small all-gather of bytes) and map the peers' buffers."""
    mine = torch.frombuffer(bytearray(rank_obj.h.fcg_slab_ipc_export()), dtype=torch.uint8).clone()
    if comm.native_a2a:
        mine = mine.to(rank_obj.xch.device)
    parts = [torch.empty_like(mine) for _ in range(comm.world)]
    comm.dist.all_gather(parts, mine)
    rank_obj.h.fcg_slab_ipc_open(b"".join(bytes(p.cpu().numpy().tobytes()) for p in parts))
    rank_obj.peers = True


def _operator_round_trip(ranks, comm, energy=False):
    """S (row transforms of the own rows) -> columns -> S (ready for the inverse row transforms), on every rank.
    energy: the column pass also leaves the rank's share of sum shat |P|^2 in xch[0] (spectral search length)."""
    peers = getattr(ranks[0], "peers", False)
    if peers:
        comm.barrier([r.xch for r in ranks])         # every rank's row pass has delivered its lines into the owners' R
    else:
        comm.all_to_all([r.recv for r in ranks], [r.send for r in ranks])
    for r in ranks:                                  # on R in place: a 5-D tensor map reads the exchange layout as columns
        r.h.fcg_slab_cols_energy(r.xch) if energy else r.h.fcg_slab_cols()
    if peers:
        comm.barrier([r.xch for r in ranks])         # every rank's column pass has scattered into the owners' S
    else:
        comm.all_to_all([r.send for r in ranks], [r.recv for r in ranks])


def _set_up(ranks, comm, k, f, u, tol, maxit, spectral):
    xs = [r.xch for r in ranks]
    for r, ui in zip(ranks, u):
        r.h.fcg_slab_setup(tol, maxit)
        r.h.fcg_slab_rows_fwd(False, ui)
    _operator_round_trip(ranks, comm)
    for r, ki, fi, ui in zip(ranks, k, f, u):
        r.h.fcg_slab_rows_inv(1, ki, ui, fi, r.xch)             # r = f - A u, p := 0; xch = {r.r, f.f} of the own rows
        if spectral:
            r.h.fcg_slab_kpp0(ki, r.xch)                        # xch[2] = sum k r^2 (the first direction is p = r)
    comm.all_reduce(xs)
    for r in ranks:
        r.h.fcg_slab_scalar(0, r.xch)
        if spectral:
            r.h.fcg_slab_scalar(3, r.xch)


def _iteration(ranks, comm, k, u, spectral):
    """One CG iteration on every rank of this process.  Every kernel returns at once when the stopping decision has been taken."""
    xs = [r.xch for r in ranks]
    for r, ui in zip(ranks, u):
        r.h.fcg_slab_rows_fwd(True, ui)                         # u += alpha p (lagged), p = r + beta p, row transforms of p
    if spectral:
        # p.Ap = sum k p^2 + sum shat |P|^2 (Parseval): alpha is known once the ranks' column passes have added up their shares, so
        # the last pass applies r -= alpha q on the fly -- one pass less than the textbook order, the same two all-reduces
        _operator_round_trip(ranks, comm, energy=True)          # xch[0] = the rank's share of sum shat |P|^2
        comm.all_reduce(xs)
        for r, ki in zip(ranks, k):
            r.h.fcg_slab_scalar(4, r.xch)                       # alpha
            r.h.fcg_slab_rows_inv(2, ki, None, None, r.xch)     # r -= alpha (k o p + C p); xch = {r.r, sum k r^2, sum k r p}
        comm.all_reduce(xs)
        for r in ranks:
            r.h.fcg_slab_scalar(5, r.xch)                       # count, convergence, beta, sum k p'^2
        return
    _operator_round_trip(ranks, comm)
    for r, ki in zip(ranks, k):
        r.h.fcg_slab_rows_inv(0, ki, None, None, r.xch)         # q = k o p + C p; xch[0] = p.q of the own rows
    comm.all_reduce(xs)
    for r in ranks:
        r.h.fcg_slab_scalar(1, r.xch)                           # alpha
        r.h.fcg_slab_update_r(r.xch)                            # r -= alpha q; xch[0] = r.r of the own rows
    comm.all_reduce(xs)
    for r in ranks:
        r.h.fcg_slab_scalar(2, r.xch)                           # count, convergence, beta


def _captured_block(ranks, comm, k, u, spectral, n):
    """n iterations recorded once into a CUDA graph (stream capture on a side stream: fcg_set_stream) and kept on the first rank
    object, keyed by the buffers it was recorded for: replaying it costs one launch instead of ~10 n host calls per rank."""
    key = (tuple(x.data_ptr() for x in list(k) + list(u)), n, bool(spectral), bool(getattr(ranks[0], "peers", False)), len(ranks))
    cache = ranks[0].__dict__.setdefault("_graphs", {})
    if key in cache:
        return cache[key]
    main = torch.cuda.current_stream()
    side = torch.cuda.Stream()
    side.wait_stream(main)
    old = [r.h.stream for r in ranks]
    g = torch.cuda.CUDAGraph()
    c0 = [r.h.fcg_last_launch_count() for r in ranks]
    try:
        for r in ranks:
            r.h.fcg_set_stream(side)
        with torch.cuda.graph(g, stream=side):
            for _ in range(n):
                _iteration(ranks, comm, k, u, spectral)
    finally:
        for r, st in zip(ranks, old):
            r.h.fcg_set_stream(st)
    main.wait_stream(side)
    # the library counted the recorded launches once, as if they had run: take them off again; every replay adds them back
    per = [r.h.fcg_last_launch_count() - c for r, c in zip(ranks, c0)]
    for r, d in zip(ranks, per):
        r.replayed_launches = getattr(r, "replayed_launches", 0) - d
    cache[key] = (g, per)
    return cache[key]


def launch_count(rank_obj) -> int:
    """Kernels of libfcg that ran for this rank's last solve: the library's own count plus those inside replayed graphs."""
    return rank_obj.h.fcg_last_launch_count() + getattr(rank_obj, "replayed_launches", 0)


def slab_solve(ranks, comm, k, f, u, tol: float, maxit: int, poll_every: int = 8, spectral: bool = True, graph=None):
    """Solve A u = f with the lattice split by rows over `ranks` (all the ranks of this process: one with DistComm, G with
    LocalComm).  k, f, u: lists, one tensor of the rank's own rows each; u in: initial guess, out: solution.
    spectral: the iteration with the spectral search length (three passes, include/fcg.h), else the textbook order (four).
    graph: replay blocks of poll_every iterations from a CUDA graph recorded at the first use with these buffers (default: on
    for LocalComm; with DistComm it needs capturable collectives -- NCCL -- and is off unless asked for: not measurable on
    this one-GPU pool).  Returns (iters, rel_residual, status) -- identical on every rank."""
    if graph is None:
        graph = isinstance(comm, LocalComm)
    n = max(1, int(poll_every))
    for r in ranks:
        r.replayed_launches = 0
    _set_up(ranks, comm, k, f, u, tol, maxit, spectral)
    blocks = 0
    while True:
        done, it, rr, st = ranks[0].h.fcg_slab_poll()           # every rank holds the same scalars
        if done:
            break
        if graph and blocks >= 1:                               # (the first block runs eagerly: short solves never pay for a capture)
            g, per = _captured_block(ranks, comm, k, u, spectral, n)
            g.replay()
            for r, d in zip(ranks, per):
                r.replayed_launches += d
        else:
            for _ in range(n):
                _iteration(ranks, comm, k, u, spectral)
        blocks += 1
    for r, ui in zip(ranks, u):
        r.h.fcg_slab_finish(ui)
    for r in ranks[1:]:
        r.h.fcg_slab_poll()
    return it, rr, st
