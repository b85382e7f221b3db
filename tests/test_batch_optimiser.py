"""Batch-size optimiser.  The host-side pipeline model is pinned
on CPU against closed forms and an independent discrete-event simulation of Alg. 2's dependency
graph; on the GPU the chosen batch must be (nearly) as fast as the best of the swept ones."""
import heapq

import pytest

import paper_2509_03933_b200 as tdma


def simulate(nb, tA, tB, tC, nstreams, last_frac):
    """Independent restatement: tasks with dependencies executed by in-order queues (streams)."""
    if nstreams == 1:
        return sum((tA + tB + tC) * (last_frac if n == nb - 1 else 1.0) for n in range(nb))
    nl = nstreams - 1
    depth = nl + 2
    queues = {("lane", i): [] for i in range(nl)}
    queues[("B", 0)] = []
    deps, dur = {}, {}
    for n in range(nb + 2):                      # enqueue order of Alg. 2
        if n < nb:
            queues[("lane", n % nl)].append(("A", n))
            deps[("A", n)] = [("C", n - depth)] if n >= depth else []
        if 0 <= n - 1 < nb:
            queues[("B", 0)].append(("B", n - 1))
            deps[("B", n - 1)] = [("A", n - 1)]
        if 0 <= n - 2 < nb:
            queues[("lane", (n - 2) % nl)].append(("C", n - 2))
            deps[("C", n - 2)] = [("B", n - 2)]
    for (s, n) in deps:
        dur[(s, n)] = {"A": tA, "B": tB, "C": tC}[s] * (last_frac if n == nb - 1 else 1.0)
    done, clock = {}, {q: 0.0 for q in queues}
    heads = {q: 0 for q in queues}
    progress = True
    while progress:
        progress = False
        for q, items in queues.items():
            while heads[q] < len(items) and all(d in done for d in deps[items[heads[q]]]):
                t = items[heads[q]]
                start = max([clock[q]] + [done[d] for d in deps[t]])
                done[t] = clock[q] = start + dur[t]
                heads[q] += 1
                progress = True
    assert len(done) == 3 * nb
    return max(done.values())


@pytest.mark.parametrize("nb", [1, 2, 3, 7, 64])
@pytest.mark.parametrize("nstreams", [1, 2, 3, 4])
@pytest.mark.parametrize("times", [(1.0, 0.1, 0.5), (0.2, 1.0, 0.1), (1.0, 1.0, 1.0), (0.3, 0.0, 0.7)])
def test_model_matches_event_simulation(nb, nstreams, times):
    for last in (1.0, 0.25):
        got = tdma.tdma_pipeline_model(nb, *times, nstreams, last)
        assert got == pytest.approx(simulate(nb, *times, nstreams, last), rel=1e-12, abs=1e-12)


def test_model_closed_forms():
    # one batch: nothing overlaps
    assert tdma.tdma_pipeline_model(1, 3.0, 2.0, 1.0, 2, 1.0) == pytest.approx(6.0)
    # stage B negligible, 2 streams: the A+C lane is the critical path
    assert tdma.tdma_pipeline_model(10, 2.0, 0.0, 1.0, 2, 1.0) == pytest.approx(30.0)
    # stage B dominant: A(0), then nb B's back to back, then C(nb-1)
    assert tdma.tdma_pipeline_model(10, 1.0, 5.0, 1.0, 2, 1.0) == pytest.approx(1.0 + 50.0 + 1.0)
    # sequential order
    assert tdma.tdma_pipeline_model(4, 1.0, 2.0, 3.0, 1, 0.5) == pytest.approx(3 * 6.0 + 3.0)
    # bad arguments
    assert tdma.tdma_pipeline_model(0, 1, 1, 1, 2, 1.0) < 0
    assert tdma.tdma_pipeline_model(3, 1, 1, 1, 2, 0.0) < 0


@pytest.mark.gpu
def test_autotune_picks_a_near_optimal_batch():
    import torch
    import tdma_inputs
    dev = torch.device("cuda:0")
    w = tdma_inputs.make_workload("cfg2_poisson", device=dev)
    x = torch.empty_like(w.d)
    cands = [1, 2, 4, 8, 16, 32, 64]
    best, est = tdma.tdma_plan_autotune(w.nx, w.ny, w.nz, w.P, cands, w.a, w.b, w.c, w.d, x, nstreams=2)
    assert best in cands and all(e > 0 for e in est)
    swept = {}
    for bz in cands:
        with tdma.Plan(w.nx, w.ny, w.nz, w.P, bz, variant=tdma.TDMA_VARIANT_PIPELINED, nstreams=2) as plan:
            for _ in range(3):
                plan.solve(w.a, w.b, w.c, w.d, x)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(5):
                plan.solve(w.a, w.b, w.c, w.d, x)
            e1.record()
            torch.cuda.synchronize()
            swept[bz] = e0.elapsed_time(e1) / 5
    # the paper's criterion is the trend, not the absolute time (PAPER.md:4.2.3): the chosen batch
    # must be within 15 % of the best swept one, and the estimates must rank bz = 1 as the worst
    assert swept[best] <= 1.15 * min(swept.values()), (best, swept, est)
    assert est[0] == max(est)
