"""SURVEY 8(f) f4, host side: the y-slab driver (paper_2509_03933_b200/yslab.py) with TWO gloo ranks on
the CPU.  The rank-local stages are the numpy stand-in of tests/yslab_standin.py (same buffer
contract as the C ABI's tdma_slab_stage_*), so what is tested here is the driver: buffer sizes,
the two all-to-alls per batch with even distribution of the lines, the remainder
batch, and the enqueue order of Alg. 2.  The result is compared
with the whole-line Thomas oracle on the undivided system."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r'''
import os, sys, json
import numpy as np, torch, torch.distributed as dist
sys.path.insert(0, %(root)r); sys.path.insert(0, os.path.join(%(root)r, "tests"))
import oracle, tdma_inputs
from yslab_standin import NumpySlabStages
from paper_2509_03933_b200.yslab import YSlabSolver
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
nx, ny, nz, P_local, batch = %(nx)d, %(ny)d, %(nz)d, %(P)d, %(batch)d
a, b, c, d = tdma_inputs.dominant_random(nx, ny, nz, 11)          # the undivided system, same bits on every rank
nyl = ny // world
sl = slice(rank * nyl, (rank + 1) * nyl)
loc = [t[:, sl, :].contiguous() for t in (a, b, c, d)]
x = torch.full_like(loc[3], float("nan"))
st = NumpySlabStages(nx, nyl, nz, P_local, batch, rank, world)
st.bind_inputs(*loc)

class FileExchange:
    # peer-mode plumbing for CPU ranks: every rank's buffer is a file mapped by all ranks
    def __init__(self, folder):
        self.folder, self.count, self.bufs, self.key = folder, 0, {}, {}
    def alloc(self, n):
        idx, self.count = self.count, self.count + 1
        path = lambda q: os.path.join(self.folder, "buf%%d_rank%%d" %% (idx, q))
        own = np.memmap(path(rank), dtype=np.float64, mode="w+", shape=(n,))
        own[:] = np.nan
        own.flush()
        dist.barrier()
        self.bufs[idx] = [torch.from_numpy(np.memmap(path(q), dtype=np.float64, mode="r+", shape=(n,))) for q in range(world)]
        t = self.bufs[idx][rank]
        self.key[t.data_ptr()] = idx
        return t
    def peers(self, t):
        return self.bufs[self.key[t.data_ptr()]]
    def barrier(self):
        dist.barrier()

exchange = FileExchange(%(peer_dir)r) if %(peer_dir)r else None
solver = YSlabSolver(nx, nyl, nz, P_local, batch, stages=st, exchange=exchange)
solver.solve(*loc, x)
ref = oracle.solve_y(*[t.numpy() for t in (a, b, c, d)])[:, sl, :]
err = float(oracle.normwise_error(np.ascontiguousarray(x.numpy()), np.ascontiguousarray(ref)).max())
print(json.dumps({"rank": rank, "err": err, "log": solver.log, "bytes": solver.exchange_bytes(0),
                  "nb": st.nb, "finite": bool(np.isfinite(x.numpy()).all())}))
dist.destroy_process_group()
'''


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _run(world, peer_dir="", **kw):
    port = _free_port()
    code = WORKER % dict(root=ROOT, peer_dir=peer_dir, **kw)
    procs = []
    for r in range(world):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(world),
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), OMP_NUM_THREADS="1")
        procs.append(subprocess.Popen([sys.executable, "-c", code], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True, cwd=ROOT))
    outs = [p.communicate(timeout=300) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e[-2000:]
    return sorted((json.loads(o.strip().splitlines()[-1]) for o, _ in outs), key=lambda r: r["rank"])


@pytest.mark.timeout(400)
@pytest.mark.parametrize("peer", [False, True], ids=["all_to_all", "peer_stores"])
@pytest.mark.parametrize("P_local,batch", [(1, 2), (2, 0), (4, 3)])
def test_yslab_driver_two_gloo_ranks_matches_whole_line_thomas(P_local, batch, peer, tmp_path):
    """peer_stores: the driver's peer mode -- no all-to-all, the stages store into the other rank's
    receive ring (files mapped by both ranks), one barrier per exchange; same result, same order."""
    nx, ny, nz = 6, 32, 7
    recs = _run(2, nx=nx, ny=ny, nz=nz, P=P_local, batch=batch, peer_dir=str(tmp_path) if peer else "")
    bz = nz if batch == 0 else batch
    nb = (nz + bz - 1) // bz
    for r in recs:
        assert r["finite"] and r["err"] <= 1e-11, r["err"]
        assert r["nb"] == nb
        # 6 values out, 2 back per (line, local partition): 48 and 16 bytes (G7)
        lb = nx * bz
        assert r["bytes"] == [48 * P_local * lb, 16 * P_local * lb]
        # Alg. 2 order: iteration n enqueues A(n), A2B(n), B(n-1), B2C(n-1), C(n-2)
        expect = []
        for n in range(nb + 2):
            if n < nb:
                expect += [["A", n], ["A2B", n]]
            if 0 <= n - 1 < nb:
                expect += [["B", n - 1], ["B2C", n - 1]]
            if 0 <= n - 2 < nb:
                expect.append(["C", n - 2])
        assert r["log"] == expect


def test_standin_reduced_rows_hold_for_the_true_solution():
    """The stand-in itself: its two boundary equations per partition are satisfied by the
    whole-line solution (pin of the test infrastructure, independent of any kernel)."""
    import oracle
    from yslab_standin import reduced_rows
    rng = np.random.default_rng(3)
    n, m = 24, 6
    a, c = rng.uniform(-1, 1, n), rng.uniform(-1, 1, n)
    b = 2.5 + rng.uniform(0, 1, n)
    d = rng.normal(size=n)
    x = np.array(oracle.thomas_line(a, b, c, d))
    for p in range(n // m):
        r = slice(p * m, (p + 1) * m)
        fa, fc, fd, pa, pc, pd = reduced_rows(a[r], b[r], c[r], d[r], p == 0, p == n // m - 1)
        xp = x[p * m - 1] if p > 0 else 0.0
        xn = x[(p + 1) * m] if p < n // m - 1 else 0.0
        assert abs(fa * xp + x[p * m] + fc * x[(p + 1) * m - 1] - fd) <= 1e-13
        assert abs(pa * x[p * m] + x[(p + 1) * m - 1] + pc * xn - pd) <= 1e-13
