"""y-slab decomposition over several GPUs: the paper's own multi-GPU
setting ("the domain is decomposed along the y-direction"; PAPER.md:106 the
all-to-all with even distribution; Alg. 2, the batch pipeline).

One process per GPU.  Rank r owns rows ``r*ny_local .. (r+1)*ny_local-1`` of every line.  The
rank-local stages are the library's kernels (``tdma_slab_stage_a / _b / _c`` of include/tdma.h); this
module is the plumbing around them: buffers, streams and events, and the two exchanges per batch as
``torch.distributed.all_to_all_single`` (NCCL on GPUs; the transfers are ``48 * P_local * Lb`` bytes
out and ``16 * P_local * Lb`` bytes back per rank and batch, a few MiB, so the library collective
on its own stream is the right tool -- no arithmetic happens here).

Schedule (Alg. 2 with events instead of stream synchronisation), iteration n = 0 .. nb+1:
    A(n) on the A+C stream            -> A2B(n)   on the communication stream
    B(n-1) on the B stream            -> B2C(n-1) on the communication stream
    C(n-2) on the A+C stream
so the reduced solve and both exchanges of a batch run behind the partition stages of its
neighbours.  Ring of 3 buffer slots ("three batched systems concurrently").

Peer mode (``exchange=``): no all-to-all at all.  The receive buffers live in memory every rank can
store into (``SymmMemExchange``: torch symmetric memory, NVLink peer mappings), stage A and stage B
write every block of their output straight into its receiver's buffer (``tdma_slab_stage_a_peer`` /
``_b_peer``), so the transfer overlaps the stage tile by tile, and each exchange shrinks to one
cross-rank barrier on the communication stream.  Ring hazards need no extra edges: A(n) follows
C(n-3) on its stream, C(n-3) waited for the barrier behind every rank's B(n-3), so recv[slot] is
free on every rank when A(n) stores into it; likewise every rank's A(n) follows its C(n-3), and
B(n) waits for the barrier behind all A(n), so yrecv[slot] is free when B(n) stores into it.

UNMEASURED ON HARDWARE with more than one GPU: this container and its GPU box have one device.
What is tested: the stages and their buffer layouts on one B200 with the ranks' exchanges emulated
by tensor permutation (tests/test_gpu_yslab.py), and this driver with two ``gloo`` ranks on the
CPU against a stand-in for the stages (tests/test_yslab_cpu.py).
"""
from __future__ import annotations

from typing import List, Optional, Tuple

import torch

from . import binding as _b

DEPTH = 3


class CudaSlabStages:
    """The rank-local stages through the C ABI (device buffers, CUDA streams)."""

    def __init__(self, nx: int, ny_local: int, nz: int, P_local: int, batch: int, rank: int, nranks: int,
                 pdd: bool = False):
        self.pdd = pdd      # stage B = PDD: 2 x 2 interface systems, an approximation
        self.nx, self.ny, self.nz, self.P, self.rank, self.nranks = nx, ny_local, nz, P_local, rank, nranks
        self.handle = _b.tdma_slab_create(nx, ny_local, nz, P_local, batch, rank, nranks)
        self.P = _b.tdma_slab_get(self.handle, _b.TDMA_SLAB_PLOCAL)     # the partitions actually exchanged
        self.tma = bool(_b.tdma_slab_get(self.handle, _b.TDMA_SLAB_TMA))
        self.nb = _b.tdma_slab_get(self.handle, _b.TDMA_SLAB_NB)
        self.bz = _b.tdma_slab_get(self.handle, _b.TDMA_SLAB_BATCH)
        self.device = torch.device("cuda", torch.cuda.current_device())

    def batch_lines(self, n: int) -> Tuple[int, int]:
        """(Lb, Ls) of batch n: its lines and every rank's share of them."""
        slices = min(self.bz, self.nz - n * self.bz)
        lb = self.nx * slices
        return lb, lb // self.nranks

    def stage_a(self, n, a, b, c, d, send, stream=None):
        _b.tdma_slab_stage_a(self.handle, n, a, b, c, d, send, stream)

    def stage_b(self, n, recv, yout, stream=None):
        (_b.tdma_slab_stage_b_pdd if self.pdd else _b.tdma_slab_stage_b)(self.handle, n, recv, yout, stream)

    def stage_c(self, n, yrecv, x, stream=None):
        _b.tdma_slab_stage_c(self.handle, n, yrecv, x, stream)

    # stages fused with their exchange: the output goes straight into the receivers' buffers
    def set_peers(self, slot, recv_of_rank, yrecv_of_rank):
        _b.tdma_slab_set_peers(self.handle, slot, recv_of_rank, yrecv_of_rank)

    def stage_a_peer(self, n, a, b, c, d, stream=None):
        _b.tdma_slab_stage_a_peer(self.handle, n, a, b, c, d, stream)

    def stage_b_peer(self, n, recv, stream=None):
        _b.tdma_slab_stage_b_peer(self.handle, n, recv, self.pdd, stream)

    def close(self):
        if self.handle:
            _b.tdma_slab_destroy(self.handle)
            self.handle = 0


class LocalExchange:
    """Peer-mode plumbing of a single rank: its own buffers, nothing to wait for."""

    def __init__(self, device):
        self.device = device

    def alloc(self, n: int) -> torch.Tensor:
        return torch.empty(n, dtype=torch.float64, device=self.device)

    def peers(self, t: torch.Tensor):
        return [t]

    def barrier(self):
        pass


class SymmMemExchange:
    """Peer-mode plumbing over torch symmetric memory (one process per GPU, NVLink peer mappings):
    ``alloc`` is collective and returns this rank's buffer, ``peers`` the device addresses of every
    rank's copy, ``barrier`` a device-side barrier over all ranks on the current stream.
    UNMEASURED: needs more than one GPU."""

    def __init__(self, group=None):
        import torch.distributed as dist
        import torch.distributed._symmetric_memory as symm
        self.symm, self.group = symm, group if group is not None else dist.group.WORLD
        self.device = torch.device("cuda", torch.cuda.current_device())
        self.handles = {}
        self.first = None

    def alloc(self, n: int) -> torch.Tensor:
        t = self.symm.empty(n, dtype=torch.float64, device=self.device)
        h = self.symm.rendezvous(t, self.group)
        self.handles[t.data_ptr()] = h
        self.first = self.first or h
        return t

    def peers(self, t: torch.Tensor):
        return [int(p) for p in self.handles[t.data_ptr()].buffer_ptrs]

    def barrier(self):
        self.first.barrier(channel=0)


class YSlabSolver:
    """Pipelined y-slab solve of one rank.  ``stages``: the rank-local stages (default: the CUDA
    kernels through the C ABI); ``group``: a torch.distributed process group (None = default group;
    with no initialised process group a single rank runs alone and the exchange is a local copy);
    ``exchange``: None = the two all-to-alls per batch; an object with ``alloc / peers / barrier``
    (``SymmMemExchange``, ``LocalExchange``) = peer mode, see the module docstring."""

    def __init__(self, nx: int, ny_local: int, nz: int, P_local: int = 1, batch: int = 0, group=None,
                 stages=None, pdd: bool = False, exchange=None):
        import torch.distributed as dist
        self.dist = dist if dist.is_available() and dist.is_initialized() else None
        self.group = group
        self.rank = self.dist.get_rank(group) if self.dist else 0
        self.nranks = self.dist.get_world_size(group) if self.dist else 1
        self.stages = stages if stages is not None else CudaSlabStages(nx, ny_local, nz, P_local, batch,
                                                                       self.rank, self.nranks, pdd=pdd)
        self.P = P_local = getattr(self.stages, "P", P_local)
        self.device = self.stages.device
        self.cuda = self.device.type == "cuda"
        lb, ls = self.stages.batch_lines(0)
        mk = lambda n: [torch.empty(n, dtype=torch.float64, device=self.device) for _ in range(DEPTH)]
        self.exchange = exchange
        if exchange is None:
            self.send, self.recv = mk(self.nranks * P_local * 6 * ls), mk(self.nranks * P_local * 6 * ls)
            self.yout, self.yrecv = mk(self.nranks * 2 * P_local * ls), mk(self.nranks * 2 * P_local * ls)
        else:       # receive rings only, in memory the other ranks store into (same allocation order on every rank)
            self.recv = [exchange.alloc(self.nranks * P_local * 6 * ls) for _ in range(DEPTH)]
            self.yrecv = [exchange.alloc(self.nranks * 2 * P_local * ls) for _ in range(DEPTH)]
            for slot in range(DEPTH):
                self.stages.set_peers(slot, exchange.peers(self.recv[slot]), exchange.peers(self.yrecv[slot]))
            exchange.barrier()      # every rank's table is set before anyone stores
        self.log: List[Tuple[str, int]] = []          # (operation, batch) in enqueue order of the last solve
        if self.cuda:
            self.s_b, self.s_comm = torch.cuda.Stream(), torch.cuda.Stream()
            ev = lambda: [torch.cuda.Event() for _ in range(DEPTH)]
            self.ev_a, self.ev_x1, self.ev_b, self.ev_x2, self.ev_c = ev(), ev(), ev(), ev(), ev()

    def exchange_bytes(self, n: int = 0) -> Tuple[int, int]:
        """Bytes this rank sends in A2B and in B2C of batch n (6 values out, 2 back)."""
        lb, ls = self.stages.batch_lines(n)
        return 8 * self.nranks * self.P * 6 * ls, 8 * self.nranks * 2 * self.P * ls

    def _all_to_all(self, out: torch.Tensor, inp: torch.Tensor):
        if self.dist is None or self.nranks == 1:
            out.copy_(inp)
        else:
            self.dist.all_to_all_single(out, inp, group=self.group)

    def solve(self, a, b, c, d, x):
        """Enqueue the whole slab solve; on CUDA the caller's current stream sees x when it returns
        (the internal streams are joined back into it)."""
        st, nb = self.stages, self.stages.nb
        self.log = []
        if self.cuda:
            s_ac = torch.cuda.current_stream()
            fork = torch.cuda.Event()
            fork.record(s_ac)
            self.s_b.wait_event(fork)
            self.s_comm.wait_event(fork)
        for n in range(nb + 2):
            if n < nb:                                    # stage A(n), then A2B(n)
                slot = n % DEPTH
                lb, ls = st.batch_lines(n)
                n6 = self.nranks * self.P * 6 * ls
                if self.exchange is not None:             # stage A stores into the receivers: A2B = a barrier
                    if self.cuda:
                        st.stage_a_peer(n, a, b, c, d, s_ac)
                        self.ev_a[slot].record(s_ac)
                        self.s_comm.wait_event(self.ev_a[slot])
                        with torch.cuda.stream(self.s_comm):
                            self.exchange.barrier()
                        self.ev_x1[slot].record(self.s_comm)
                    else:
                        st.stage_a_peer(n, a, b, c, d)
                        self.exchange.barrier()
                elif self.cuda:
                    if n >= DEPTH:
                        s_ac.wait_event(self.ev_x1[slot])      # send[slot] was read by A2B(n - DEPTH)
                    st.stage_a(n, a, b, c, d, self.send[slot], s_ac)
                    self.ev_a[slot].record(s_ac)
                    self.s_comm.wait_event(self.ev_a[slot])
                    if n >= DEPTH:
                        self.s_comm.wait_event(self.ev_b[slot])  # recv[slot] was read by B(n - DEPTH)
                    with torch.cuda.stream(self.s_comm):
                        self._all_to_all(self.recv[slot][:n6], self.send[slot][:n6])
                    self.ev_x1[slot].record(self.s_comm)
                else:
                    st.stage_a(n, a, b, c, d, self.send[slot])
                    self._all_to_all(self.recv[slot][:n6], self.send[slot][:n6])
                self.log += [("A", n), ("A2B", n)]
            q = n - 1
            if 0 <= q < nb:                               # stage B(n-1), then B2C(n-1)
                slot = q % DEPTH
                lb, ls = st.batch_lines(q)
                n2 = self.nranks * 2 * self.P * ls
                if self.exchange is not None:             # stage B stores into the receivers: B2C = a barrier
                    if self.cuda:
                        self.s_b.wait_event(self.ev_x1[slot])
                        st.stage_b_peer(q, self.recv[slot], self.s_b)
                        self.ev_b[slot].record(self.s_b)
                        self.s_comm.wait_event(self.ev_b[slot])
                        with torch.cuda.stream(self.s_comm):
                            self.exchange.barrier()
                        self.ev_x2[slot].record(self.s_comm)
                    else:
                        st.stage_b_peer(q, self.recv[slot])
                        self.exchange.barrier()
                elif self.cuda:
                    self.s_b.wait_event(self.ev_x1[slot])
                    if q >= DEPTH:
                        self.s_b.wait_event(self.ev_x2[slot])    # yout[slot] was read by B2C(q - DEPTH)
                    st.stage_b(q, self.recv[slot], self.yout[slot], self.s_b)
                    self.ev_b[slot].record(self.s_b)
                    self.s_comm.wait_event(self.ev_b[slot])
                    if q >= DEPTH:
                        self.s_comm.wait_event(self.ev_c[slot])  # yrecv[slot] was read by C(q - DEPTH)
                    with torch.cuda.stream(self.s_comm):
                        self._all_to_all(self.yrecv[slot][:n2], self.yout[slot][:n2])
                    self.ev_x2[slot].record(self.s_comm)
                else:
                    st.stage_b(q, self.recv[slot], self.yout[slot])
                    self._all_to_all(self.yrecv[slot][:n2], self.yout[slot][:n2])
                self.log += [("B", q), ("B2C", q)]
            q = n - 2
            if 0 <= q < nb:                               # stage C(n-2)
                slot = q % DEPTH
                if self.cuda:
                    s_ac.wait_event(self.ev_x2[slot])
                    st.stage_c(q, self.yrecv[slot], x, s_ac)
                    self.ev_c[slot].record(s_ac)
                else:
                    st.stage_c(q, self.yrecv[slot], x)
                self.log.append(("C", q))
        if self.cuda:
            join_b, join_c = torch.cuda.Event(), torch.cuda.Event()
            join_b.record(self.s_b)
            join_c.record(self.s_comm)
            s_ac.wait_event(join_b)
            s_ac.wait_event(join_c)
        return x

    def close(self):
        if hasattr(self.stages, "close"):
            self.stages.close()

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()
