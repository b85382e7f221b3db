"""tdma_solve_static (include/tdma.h): the allocation-free entry point, whose scratch is a file-scope
__device__ array of the library, against the existing path (a PIPELINED plan: the same stage
kernels with plan-owned scratch) and against the oracle, on two calls in a row that share the
array.  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest
import torch

import oracle
import tdma_inputs
import paper_2509_03933_b200 as tdma

pytestmark = pytest.mark.gpu
TOL_E = 1e-11


def dev():
    return torch.device("cuda:0")


def plan_solve(a, b, c, d, P):
    nz, ny, nx = a.shape
    x = torch.full_like(d, float("nan"))
    with tdma.Plan(nx, ny, nz, P, 0, variant=tdma.TDMA_VARIANT_PIPELINED) as plan:
        plan.solve(a, b, c, d, x)
        torch.cuda.synchronize()
    return x


def check(a, b, c, d, x, x_plan):
    an, bn, cn, dn, xn = [t.cpu().numpy() for t in (a, b, c, d, x)]
    assert np.isfinite(xn).all()
    assert oracle.normwise_error(xn, x_plan.cpu().numpy()).max() <= TOL_E
    assert oracle.normwise_error(xn, oracle.solve_y(an, bn, cn, dn)).max() <= TOL_E


def test_two_calls_in_a_row_match_the_plan_path_and_the_oracle():
    """Two different systems of different shapes, one call right after the other on the same stream
    (the second call finds the first one's contents in the static array), no allocation in between:
    every tensor exists before the first call.  The second shape spans several batches of the static
    array (3 * 8 * 512 * 256 * 40 bytes > 32 MiB) with a ragged last one."""
    dv = dev()
    cases = [((7, 64, 96), 4, 71), ((40, 256, 512), 8, 72)]
    data = []
    for (nz, ny, nx), P, seed in cases:
        a, b, c, d = tdma_inputs.dominant_random(nx, ny, nz, seed, dv)
        data.append((a, b, c, d, torch.full_like(d, float("nan")), P, plan_solve(a, b, c, d, P)))
    a, b, c, d, x, P, _ = data[0]
    tdma.tdma_solve_static(a.shape[2], a.shape[1], a.shape[0], P, a, b, c, d, x)   # first use on this device: loads the kernels
    x.fill_(float("nan"))
    torch.cuda.synchronize()
    before, free_before = torch.cuda.memory_allocated(), torch.cuda.mem_get_info()[0]
    for a, b, c, d, x, P, _ in data:
        nz, ny, nx = a.shape
        tdma.tdma_solve_static(nx, ny, nz, P, a, b, c, d, x)
    torch.cuda.synchronize()
    # no device memory was taken: a plan for the second shape would hold > 30 MB of scratch
    assert torch.cuda.memory_allocated() == before and free_before - torch.cuda.mem_get_info()[0] < (1 << 20)
    for a, b, c, d, x, P, x_plan in data:
        check(a, b, c, d, x, x_plan)
        assert torch.equal(x, x_plan)          # same kernels, same arithmetic: the same bits


def test_same_system_twice_and_in_place():
    """The same call twice gives the same bits (nothing depends on what the array held), also with
    x aliasing d; Poisson lines of cfg 2 (weakly dominant, pinned mean mode)."""
    w = tdma_inputs.make_workload("cfg2_poisson", device=dev(), nz=12)
    x_plan = plan_solve(w.a, w.b, w.c, w.d, w.P)
    x1, x2 = torch.full_like(w.d, float("nan")), w.d.clone()
    tdma.tdma_solve_static(w.nx, w.ny, w.nz, w.P, w.a, w.b, w.c, w.d, x1)
    tdma.tdma_solve_static(w.nx, w.ny, w.nz, w.P, w.a, w.b, w.c, x2, x2)
    torch.cuda.synchronize()
    assert torch.equal(x1, x2) and torch.equal(x1, x_plan)
    an, bn, cn, dn, xn = [t.cpu().numpy() for t in (w.a, w.b, w.c, w.d, x1)]
    assert oracle.normwise_error(xn, oracle.solve_y(an, bn, cn, dn, "ld")).max() <= TOL_E


def test_shapes_beyond_the_static_array_are_refused():
    t = torch.zeros(16, dtype=torch.float64, device=dev())
    with pytest.raises(tdma.TdmaError) as e:                 # one 2048 x 1024 slice: 51 MB of scratch
        tdma.tdma_solve_static(2048, 1024, 1, 16, t, t, t, t, t)
    assert e.value.status == tdma.TDMA_ERR_UNSUPPORTED and "TDMA_STATIC_SCRATCH_BYTES" in str(e.value)
    with pytest.raises(tdma.TdmaError) as e:
        tdma.tdma_solve_static(16, 30, 1, 4, t, t, t, t, t)  # 30 rows, 4 partitions
    assert e.value.status == tdma.TDMA_ERR_INVALID_ARG
    with pytest.raises(tdma.TdmaError):
        tdma.tdma_solve_static(16, 32, 1, 4, t, t, t, 0, t)  # NULL array
