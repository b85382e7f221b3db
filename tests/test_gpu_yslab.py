"""SURVEY 8(f) f4 on ONE B200: the rank-local stages of the y-slab decomposition
(tdma_slab_stage_a / _b / _c through the C ABI) for all ranks of an emulated job, run one after
the other in this process with the two all-to-alls done by tensor permutation (nothing here waits
on another launch).  x is compared with the whole-line Thomas oracle on the undivided system, the
exchange buffers with the Schur-complement stand-in of tests/yslab_standin.py.  The driver
(yslab.YSlabSolver) is run as a single rank to exercise its streams and events on hardware.
More than one GPU: unmeasured (the box has one)."""
import numpy as np
import pytest
import torch

import oracle
import tdma_inputs
import paper_2509_03933_b200 as tdma
from paper_2509_03933_b200.yslab import YSlabSolver, CudaSlabStages, LocalExchange
from yslab_standin import reduced_rows

pytestmark = pytest.mark.gpu
TOL_E = 1e-11


def dev():
    return torch.device("cuda:0")


def emulate(a, b, c, d, nranks, P_local, batch, keep=None, pdd=False, info=None):
    """All ranks' stages in sequence; returns x of the undivided slab."""
    nz, ny, nx = a.shape
    nyl = ny // nranks
    loc = [[t[:, r * nyl:(r + 1) * nyl, :].contiguous() for t in (a, b, c, d)] for r in range(nranks)]
    xs = [torch.full_like(loc[r][3], float("nan")) for r in range(nranks)]
    st = [CudaSlabStages(nx, nyl, nz, P_local, batch, r, nranks, pdd=pdd) for r in range(nranks)]
    P_local = st[0].P                   # the partitions per rank actually exchanged (TMA stages: the tiling's)
    assert all(s.P == P_local for s in st)
    if info is not None:
        info.update(P=P_local, tma=st[0].tma)
    try:
        for n in range(st[0].nb):
            lb, ls = st[0].batch_lines(n)
            send = torch.full((nranks, nranks, P_local, 6, ls), float("nan"), dtype=torch.float64, device=a.device)
            for r in range(nranks):
                st[r].stage_a(n, *loc[r], send[r])
            recv = send.transpose(0, 1).contiguous()          # recv[q][src] = send[src][dest = q]
            yout = torch.full((nranks, nranks, 2 * P_local, ls), float("nan"), dtype=torch.float64, device=a.device)
            for q in range(nranks):
                st[q].stage_b(n, recv[q], yout[q])
            yrecv = yout.transpose(0, 1).contiguous()         # yrecv[r][src] = yout[src][dest = r]
            for r in range(nranks):
                st[r].stage_c(n, yrecv[r], xs[r])
            torch.cuda.synchronize()
            if keep is not None:
                keep.append((n, send.cpu().numpy(), yout.cpu().numpy(), P_local))
    finally:
        for s in st:
            s.close()
    return torch.cat(xs, dim=1)


@pytest.mark.parametrize("nranks,P_local,batch", [(2, 1, 0), (2, 4, 3), (4, 2, 2), (8, 1, 4), (4, 4, 0)])
def test_emulated_ranks_match_whole_line_thomas(nranks, P_local, batch):
    nx, ny, nz = 64, 256, 7
    a, b, c, d = tdma_inputs.dominant_random(nx, ny, nz, 41, dev())
    x = emulate(a, b, c, d, nranks, P_local, batch)
    an, bn, cn, dn, xn = [t.cpu().numpy() for t in (a, b, c, d, x)]
    assert np.isfinite(xn).all()
    assert oracle.normwise_error(xn, oracle.solve_y(an, bn, cn, dn)).max() <= TOL_E


def test_poisson_slab_over_four_emulated_ranks():
    """cfg-2 coefficients (weakly dominant, pinned mean mode), 4 ranks x 64 rows: long-double reference."""
    w = tdma_inputs.make_workload("cfg2_poisson", device=dev(), nz=8)
    x = emulate(w.a, w.b, w.c, w.d, 4, 2, 4)
    an, bn, cn, dn, xn = [t.cpu().numpy() for t in (w.a, w.b, w.c, w.d, x)]
    assert oracle.normwise_error(xn, oracle.solve_y(an, bn, cn, dn, "ld")).max() <= TOL_E


@pytest.mark.parametrize("nranks,P_local", [(4, 1), (2, 2)])
def test_pdd_over_emulated_ranks(nranks, P_local):
    """PDD reduced solve across emulated ranks: parity with oracle.solve_y_pdd for
    nranks * P_local partitions (both drop the far spike ends), and -- 64-row partitions of a
    strictly dominant system -- agreement with the exact solve far below the tolerance."""
    nx, ny, nz = 32, 256, 4
    a, b, c, d = tdma_inputs.dominant_random(nx, ny, nz, 53, dev())
    info = {}
    x = emulate(a, b, c, d, nranks, P_local, 2, pdd=True, info=info)
    an, bn, cn, dn, xn = [t.cpu().numpy() for t in (a, b, c, d, x)]
    assert oracle.normwise_error(xn, oracle.solve_y_pdd(an, bn, cn, dn, nranks * info["P"])).max() <= TOL_E
    assert oracle.normwise_error(xn, oracle.solve_y(an, bn, cn, dn)).max() <= TOL_E


@pytest.mark.parametrize("nx,ny,want_tma", [(64, 256, True), (64, 1024, True), (63, 256, False), (64, 120, False)])
def test_tma_staged_stages_are_used_when_the_slab_tiles(nx, ny, want_tma):
    """4 ranks: slabs of 64 / 256 rows tile for the TMA kernel (stage A / C staged on chip, no scratch
    ring); odd nx or 30 rows per rank fall back to the one-thread-per-(line, partition) kernels.  Same
    result either way."""
    nz = 4
    a, b, c, d = tdma_inputs.dominant_random(nx, ny, nz, 59, dev())
    info = {}
    x = emulate(a, b, c, d, 4, 2, 4, info=info)
    assert info["tma"] == want_tma
    an, bn, cn, dn, xn = [t.cpu().numpy() for t in (a, b, c, d, x)]
    assert oracle.normwise_error(xn, oracle.solve_y(an, bn, cn, dn)).max() <= TOL_E


def test_exchange_buffers_hold_the_schur_complement_rows():
    """Stage A's send buffer (layout [dest][P][6][Ls]) against the definition of the reduced rows, and
    stage B's yout against the oracle's x at the partition ends."""
    nx, ny, nz, nranks, P_local = 16, 48, 3, 2, 3
    a, b, c, d = tdma_inputs.dominant_random(nx, ny, nz, 43, dev())
    keep = []
    emulate(a, b, c, d, nranks, P_local, 2, keep)
    an, bn, cn, dn = [t.cpu().numpy() for t in (a, b, c, d)]
    ref = oracle.solve_y(an, bn, cn, dn)
    bz = 2
    for n, send, yout, P_local in keep:
        m = ny // nranks // P_local
        ls = send.shape[-1]
        lb = ls * nranks
        for l in range(0, lb, 5):
            k, i = n * bz + l // nx, l % nx
            for r in range(nranks):
                for p in range(P_local):
                    pg = r * P_local + p
                    rows = slice(pg * m, (pg + 1) * m)
                    want = reduced_rows(an[k, rows, i], bn[k, rows, i], cn[k, rows, i], dn[k, rows, i],
                                        pg == 0, pg == nranks * P_local - 1)
                    got = send[r, l // ls, p, :, l % ls]
                    assert np.max(np.abs(got - np.array(want))) <= 1e-12
                    # yout[q = l // ls][dest = r][2p, 2p+1][l % ls] = x at the partition's ends
                    assert abs(yout[l // ls, r, 2 * p, l % ls] - ref[k, pg * m, i]) <= 1e-12
                    assert abs(yout[l // ls, r, 2 * p + 1, l % ls] - ref[k, (pg + 1) * m - 1, i]) <= 1e-12


@pytest.mark.parametrize("peer", [False, True], ids=["all_to_all", "peer_stores"])
@pytest.mark.parametrize("batch", [0, 2])
def test_driver_single_rank_streams_and_events(batch, peer):
    """YSlabSolver as one rank (the exchange degenerates to a copy; in peer mode the stages store into
    the rank's own receive ring): its three streams, the event ring and the join back into the
    caller's stream, on hardware; x read right after solve()."""
    nx, ny, nz = 128, 128, 9
    a, b, c, d = tdma_inputs.dominant_random(nx, ny, nz, 47, dev())
    x = torch.full_like(d, float("nan"))
    with YSlabSolver(nx, ny, nz, P_local=4, batch=batch, exchange=LocalExchange(dev()) if peer else None) as solver:
        for _ in range(2):
            solver.solve(a, b, c, d, x)
        xn = x.cpu().numpy()                      # same stream as the caller's: ordered after the join
    an, bn, cn, dn = [t.cpu().numpy() for t in (a, b, c, d)]
    assert oracle.normwise_error(xn, oracle.solve_y(an, bn, cn, dn)).max() <= TOL_E


def test_slab_create_rejects_bad_shapes():
    for args in [(16, 30, 4, 4, 0, 0, 2),      # 30 rows not divisible by 4 partitions
                 (16, 4, 4, 4, 0, 0, 2),       # 1 row per partition
                 (5, 32, 3, 1, 0, 0, 2),       # 15 lines per batch not divisible by 2 ranks
                 (16, 32, 4, 1, 0, 2, 2)]:     # rank out of range
        with pytest.raises(tdma.TdmaError):
            tdma.tdma_slab_create(*args)


def emulate_peer(a, b, c, d, nranks, P_local, batch, pdd=False):
    """The same job with the stages storing straight into the receivers' buffers
    (tdma_slab_set_peers + _stage_a_peer / _stage_b_peer): no send / yout buffer, no permutation.  All
    "ranks" live on this GPU, so the peer pointers are plain device pointers.  Returns x and, per batch,
    every rank's recv and yrecv buffer."""
    nz, ny, nx = a.shape
    nyl = ny // nranks
    loc = [[t[:, r * nyl:(r + 1) * nyl, :].contiguous() for t in (a, b, c, d)] for r in range(nranks)]
    xs = [torch.full_like(loc[r][3], float("nan")) for r in range(nranks)]
    st = [CudaSlabStages(nx, nyl, nz, P_local, batch, r, nranks, pdd=pdd) for r in range(nranks)]
    P = st[0].P
    lb0, ls0 = st[0].batch_lines(0)
    mk = lambda rows: [[torch.full((nranks * rows * ls0,), float("nan"), dtype=torch.float64, device=a.device)
                        for _ in range(nranks)] for _ in range(3)]
    recv, yrecv = mk(P * 6), mk(2 * P)                      # [slot][rank]
    kept = []
    try:
        for slot in range(3):
            for s in st:
                s.set_peers(slot, recv[slot], yrecv[slot])
        for n in range(st[0].nb):
            slot = n % 3
            lb, ls = st[0].batch_lines(n)
            for r in range(nranks):
                st[r].stage_a_peer(n, *loc[r])
            for q in range(nranks):
                st[q].stage_b_peer(n, recv[slot][q])
            for r in range(nranks):
                st[r].stage_c(n, yrecv[slot][r], xs[r])
            torch.cuda.synchronize()
            kept.append((n, ls, [t[:nranks * P * 6 * ls].clone() for t in recv[slot]],
                         [t[:nranks * 2 * P * ls].clone() for t in yrecv[slot]]))
    finally:
        for s in st:
            s.close()
    return torch.cat(xs, dim=1), kept, P


@pytest.mark.parametrize("pdd", [False, True], ids=["thomas", "pdd"])
@pytest.mark.parametrize("nx,ny,nranks,P_local,batch", [(64, 256, 4, 2, 3), (64, 256, 2, 4, 0), (27, 90, 3, 3, 4),
                                                        (64, 512, 8, 1, 2)])
def test_peer_stores_equal_the_all_to_all(nx, ny, nranks, P_local, batch, pdd):
    """Stage A / B fused with their exchange: every rank's recv / yrecv buffer and x are BITWISE what
    the buffered stages followed by the all-to-all (tensor permutation) produce, for the TMA-staged
    and the thread-per-line kernels, a ragged last batch included; x against the oracle."""
    nz = 7
    a, b, c, d = tdma_inputs.dominant_random(nx, ny, nz, 61, dev())
    keep = []
    x_ref = emulate(a, b, c, d, nranks, P_local, batch, keep, pdd=pdd)
    x, kept, P = emulate_peer(a, b, c, d, nranks, P_local, batch, pdd=pdd)
    assert torch.equal(x, x_ref)
    assert len(kept) == len(keep)
    for (n, send, yout, P_ref), (n2, ls, recv, yrecv) in zip(keep, kept):
        assert n == n2 and P == P_ref
        for q in range(nranks):
            want_recv = np.ascontiguousarray(send[:, q]).reshape(-1)        # recv[q][src] = send[src][dest = q]
            want_y = np.ascontiguousarray(yout[:, q]).reshape(-1)
            assert np.array_equal(recv[q].cpu().numpy(), want_recv)
            assert np.array_equal(yrecv[q].cpu().numpy(), want_y)
    an, bn, cn, dn, xn = [t.cpu().numpy() for t in (a, b, c, d, x)]
    ref = oracle.solve_y_pdd(an, bn, cn, dn, nranks * P) if pdd else oracle.solve_y(an, bn, cn, dn)
    assert oracle.normwise_error(xn, ref).max() <= TOL_E


def test_peer_stages_need_their_table():
    s = CudaSlabStages(32, 64, 2, 2, 0, 0, 2)
    try:
        t = torch.zeros(32 * 64 * 2, dtype=torch.float64, device=dev())
        with pytest.raises(tdma.TdmaError):
            s.stage_a_peer(0, t, t, t, t)
        with pytest.raises(tdma.TdmaError):
            s.set_peers(3, [t, t], [t, t])                   # slots 0..2
    finally:
        s.close()
