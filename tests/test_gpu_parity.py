"""Parity tests proper: the CUDA path (through the C ABI) against the CPU oracle, element by
element on the same seeded inputs.  Tolerances (BASELINE.json north_star):

  * strictly dominant configs (1, 4-y, 5):  E = max_lines ||x - x_or||_inf / ||x_or||_inf <= 1e-11
    and the literal residual  ||Ax - d||_inf <= 1e-12 ||d||_inf  per line;
  * weakly dominant Poisson configs (2, 3): E <= 1e-11 against the LONG-DOUBLE oracle and the
    normwise backward error ||Ax-d||_inf / (||A||_inf ||x||_inf + ||d||_inf) <= 1e-12; the literal
    residual is reported next to the oracle's own (fp64 Thomas does not meet it either on the
    lowest wavenumbers).
Residuals are evaluated on the host in long double.
"""
import numpy as np
import pytest
import torch

import oracle
import tdma_inputs
import paper_2509_03933_b200 as tdma

from test_golden import load_cfg1_golden

pytestmark = pytest.mark.gpu

TOL_E = 1e-11
TOL_RES = 1e-12
# the code paths behind tdma_solve: stage kernels + stream pipeline, the register-staged fused
# kernel, FUSED with fused_impl = auto (the TMA kernel wherever it is eligible), and the stage
# pipeline with TMA-staged stage A / C kernels (STAGED)
VARIANT_OPTS = [dict(variant=tdma.TDMA_VARIANT_PIPELINED),
                dict(variant=tdma.TDMA_VARIANT_FUSED, fused_impl=1),
                dict(variant=tdma.TDMA_VARIANT_FUSED),
                dict(variant=tdma.TDMA_VARIANT_STAGED)]
VARIANTS = [pytest.param(o, id=i) for o, i in zip(VARIANT_OPTS, ("pipelined", "fused_reg", "fused_tma", "staged"))]
TMA = dict(variant=tdma.TDMA_VARIANT_FUSED, fused_impl=2)


def dev():
    return torch.device("cuda:0")


def gpu_solve(a, b, c, d, P, batch=0, out=None, **opts):
    nz, ny, nx = a.shape
    x = torch.full_like(d, float("nan")) if out is None else out
    with tdma.Plan(nx, ny, nz, P, batch, **opts) as plan:
        plan.solve(a, b, c, d, x)
        torch.cuda.synchronize()
    return x


def to_np(*ts):
    return [t.detach().cpu().numpy() for t in ts]


def check_against_oracle(a, b, c, d, x, strictly_dominant, precision=None):
    an, bn, cn, dn, xn = to_np(a, b, c, d, x)
    assert np.isfinite(xn).all()
    prec = precision or ("f64" if strictly_dominant else "ld")
    ref = oracle.solve_y(an, bn, cn, dn, prec)
    E = oracle.normwise_error(xn, ref)
    res, dinf, xinf, ainf = oracle.residual_y(an, bn, cn, dn, xn)
    assert E.max() <= TOL_E, "normwise error %.3e" % E.max()
    bwd = res / (ainf * xinf + dinf + 1e-300)
    assert bwd.max() <= TOL_RES
    if strictly_dominant:
        assert (res <= TOL_RES * dinf).all(), "literal residual %.3e" % (res / dinf).max()
    return E.max()


# ---------------------------------------------------------------------------------------------
# BASELINE configs
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("batch", [0, 1, 24])
def test_cfg1_tiny_full(variant, batch):
    w = tdma_inputs.make_workload("cfg1_tiny", device=dev())
    x = gpu_solve(w.a, w.b, w.c, w.d, w.P, batch, **variant)
    check_against_oracle(w.a, w.b, w.c, w.d, x, True)
    xn = x.cpu().numpy()
    for i, k, ref in load_cfg1_golden():
        assert np.max(np.abs(xn[k, :, i] - ref)) <= TOL_E * np.max(np.abs(ref))


@pytest.mark.parametrize("variant", VARIANTS)
def test_cfg2_poisson_full(variant):
    w = tdma_inputs.make_workload("cfg2_poisson", device=dev())
    x = gpu_solve(w.a, w.b, w.c, w.d, w.P, w.batch, **variant)
    check_against_oracle(w.a, w.b, w.c, w.d, x, False)


@pytest.mark.parametrize("variant", VARIANTS)
def test_cfg4_adi_y_slab(variant):
    """512 x 512 x 48 slices of cfg 4 (full nx, ny, P; ragged last batch 48 = 32 + 16)."""
    w = tdma_inputs.make_workload("cfg4_adi_y", device=dev(), nz=48)
    x = gpu_solve(w.a, w.b, w.c, w.d, w.P, 32, **variant)
    check_against_oracle(w.a, w.b, w.c, w.d, x, True)


@pytest.mark.parametrize("variant", VARIANTS)
def test_cfg5_stress_slab(variant):
    """2048 x 512 x 20 slices of cfg 5 (m = 8, 128-row reduced system), batch 8 -> 8+8+4."""
    w = tdma_inputs.make_workload("cfg5_stress", device=dev(), nz=20)
    x = gpu_solve(w.a, w.b, w.c, w.d, w.P, 8, **variant, nstreams=3)
    check_against_oracle(w.a, w.b, w.c, w.d, x, True)


@pytest.mark.parametrize("variant", VARIANTS)
def test_cfg3_weak_slab(variant):
    """1024 x 1024 x 12 slices of cfg 3 starting at k = 0 (holds the pinned (0,0) mode and the
    lowest wavenumbers = the worst-conditioned lines), batch 8 -> 8 + 4."""
    w = tdma_inputs.make_workload("cfg3_weak", device=dev(), nz=12)
    x = gpu_solve(w.a, w.b, w.c, w.d, w.P, 8, **variant)
    check_against_oracle(w.a, w.b, w.c, w.d, x, False)


# ---------------------------------------------------------------------------------------------
# Full-size runs in the launch configuration bench.py times, sampled slices
# ---------------------------------------------------------------------------------------------
def _sampled_full(name, variant, batch, slices, strictly, **opts):
    """Full-size slab through one plan; `slices` are checked against the oracle one by one.  For
    FUSED plans that use a fill launch (clusters of 2 on the SMs the main launch leaves empty) the
    first, middle and last slice of the fill range are added, so both tilings are covered."""
    free, _ = torch.cuda.mem_get_info()
    spec = tdma_inputs.config_spec(name)
    need = spec["nx"] * spec["ny"] * spec["nz"] * 8 * 5 * 1.25
    if free < need:
        pytest.skip("needs %.0f GB of device memory" % (need / 1e9))
    w = tdma_inputs.make_workload(name, device=dev())
    x = torch.full_like(w.d, float("nan"))
    with tdma.Plan(w.nx, w.ny, w.nz, w.P, batch, **variant, **opts) as plan:
        plan.solve(w.a, w.b, w.c, w.d, x)
        torch.cuda.synchronize()
        fill = plan.get(tdma.TDMA_GET_FUSED_FILL) if variant["variant"] == tdma.TDMA_VARIANT_FUSED else 0
        launches = plan.get(tdma.TDMA_GET_LAUNCHES)
    assert bool(torch.isfinite(x).all())
    slices = list(slices)
    if fill > 0:
        slices += [w.nz - fill, w.nz - fill // 2 - 1, w.nz - 1]
        slices += [w.nz - fill - 1]                       # last slice of the main launch
    worst = 0.0
    for k in sorted(set(slices)):
        sl = slice(k, k + 1)
        worst = max(worst, check_against_oracle(w.a[sl], w.b[sl], w.c[sl], w.d[sl], x[sl], strictly))
    del w, x
    torch.cuda.empty_cache()
    return worst, fill, launches


@pytest.mark.parametrize("variant", VARIANTS)
def test_cfg3_full_size_sampled(variant):
    _sampled_full("cfg3_weak", variant, 32, [0, 1, 513, 1023], False)


@pytest.mark.parametrize("variant", VARIANTS)
def test_cfg5_full_size_sampled(variant):
    _sampled_full("cfg5_stress", variant, 16, [0, 777, 1023], True, nstreams=3)


@pytest.mark.parametrize("name,slices,strictly", [("cfg3_weak", [0, 1, 2, 257, 513, 900], False),
                                                  ("cfg5_stress", [0, 1, 300, 777], True)])
def test_full_size_in_the_bench_launch_configuration(name, slices, strictly):
    """Exactly what bench.py times: FUSED, batch = 0, i.e. persistent launches of 2^27 cells (128
    slices, ~250 tiles per cluster on cfg 3), each with its concurrent fill launch where clusters
    of 4 leave SMs empty; slices of main and fill ranges of several launches against the oracle."""
    worst, fill, launches = _sampled_full(name, dict(variant=tdma.TDMA_VARIANT_FUSED), 0, slices, strictly)
    assert launches == 8 * (2 if fill > 0 else 1)


# ---------------------------------------------------------------------------------------------
# Schedule invariance: per-line arithmetic does not depend on batching,
# stream count, graph capture or gather placement -> bitwise identical x
# ---------------------------------------------------------------------------------------------
def test_schedule_invariance_pipelined():
    w = tdma_inputs.make_workload("cfg1_tiny", device=dev())
    base = gpu_solve(w.a, w.b, w.c, w.d, w.P, 0, variant=tdma.TDMA_VARIANT_PIPELINED, nstreams=1)
    for batch in (1, 2, 7, 16, 64):
        for opts in (dict(nstreams=2), dict(nstreams=3), dict(nstreams=4, use_graph=-1),
                     dict(nstreams=2, separate_gather=1), dict(nstreams=1, use_graph=-1)):
            x = gpu_solve(w.a, w.b, w.c, w.d, w.P, batch, variant=tdma.TDMA_VARIANT_PIPELINED, **opts)
            assert torch.equal(x, base), (batch, opts)


def test_schedule_invariance_fused_batches():
    w = tdma_inputs.make_workload("cfg1_tiny", device=dev())
    base = gpu_solve(w.a, w.b, w.c, w.d, w.P, 0, variant=tdma.TDMA_VARIANT_FUSED)
    for batch in (1, 5, 32):
        x = gpu_solve(w.a, w.b, w.c, w.d, w.P, batch, variant=tdma.TDMA_VARIANT_FUSED)
        assert torch.equal(x, base)


@pytest.mark.parametrize("cluster,lines,leaf,top", [
    (1, 32, 0, 0), (2, 32, 0, 0), (4, 16, 0, 0), (4, 32, 0, 0), (2, 8, 0, 0),
    (1, 32, 16, 1), (1, 32, 16, 2),      # leaf = partition: no partition level
    (1, 32, 4, 1), (1, 32, 4, 2),        # 4 leaves per partition, 2P-row / 2-row top system
    (2, 32, 2, 1), (2, 32, 2, 2),        # two-row leaves (no interior)
    (4, 32, 8, 1), (4, 32, 8, 2), (2, 16, 8, 2), (4, 8, 4, 1),
])
def test_fused_cluster_shapes(cluster, lines, leaf, top):
    w = tdma_inputs.make_workload("cfg1_tiny", device=dev())
    with tdma.Plan(w.nx, w.ny, w.nz, w.P, 0, variant=tdma.TDMA_VARIANT_FUSED, fused_impl=1,
                   fused_cluster=cluster, fused_lines=lines, fused_leaf_rows=leaf, fused_top=top) as plan:
        assert plan.get(tdma.TDMA_GET_FUSED_CLUSTER) == cluster
        assert plan.get(tdma.TDMA_GET_FUSED_LINES) == lines
        if leaf:
            assert plan.get(tdma.TDMA_GET_FUSED_LEAF_ROWS) == leaf
        if top == 1:
            assert plan.get(tdma.TDMA_GET_FUSED_TOP_ROWS) == 2 * w.P
        if top == 2:
            assert plan.get(tdma.TDMA_GET_FUSED_TOP_ROWS) == 2 * cluster
        x = torch.full_like(w.d, float("nan"))
        plan.solve(w.a, w.b, w.c, w.d, x)
        torch.cuda.synchronize()
    check_against_oracle(w.a, w.b, w.c, w.d, x, True)


@pytest.mark.parametrize("cluster,top", [(8, 1), (8, 2), (16, 2)])
def test_fused_cluster8_16(cluster, top):
    P = 16 if cluster == 16 else 8
    w = tdma_inputs.make_workload("cfg1_tiny", device=dev(), P=P)
    x = gpu_solve(w.a, w.b, w.c, w.d, P, 0, variant=tdma.TDMA_VARIANT_FUSED, fused_impl=1,
                  fused_cluster=cluster, fused_lines=32, fused_top=top)
    check_against_oracle(w.a, w.b, w.c, w.d, x, True)


def test_fused_top_modes_agree_with_pipelined_to_rounding():
    """The 2P-row reduced system is a Schur complement: however the recursion is cut, the result
    is the same up to rounding (cfg 2 slab, weakly dominant lines included)."""
    w = tdma_inputs.make_workload("cfg2_poisson", device=dev(), nz=6)
    xs = [gpu_solve(w.a, w.b, w.c, w.d, w.P, 0, variant=tdma.TDMA_VARIANT_FUSED, fused_impl=1,
                    fused_top=top, fused_leaf_rows=leaf) for top, leaf in ((1, 0), (2, 0), (1, 32), (2, 4))]
    xs += [gpu_solve(w.a, w.b, w.c, w.d, w.P, 0, fused_leaf_rows=leaf, fused_cluster=cl, **TMA)
           for leaf, cl in ((0, 0), (2, 8), (16, 2), (4, 8))]
    for x in xs:
        check_against_oracle(w.a, w.b, w.c, w.d, x, False)


def _view(ptr, nbytes, shape):
    """Wrap a plan-owned device buffer as a torch tensor without copying."""
    n = int(np.prod(shape))
    assert n * 8 <= nbytes

    class _Holder:
        pass
    h = _Holder()
    h.__cuda_array_interface__ = {"shape": tuple(shape), "typestr": "<f8", "data": (ptr, False),
                                  "version": 3, "strides": None}
    return torch.as_tensor(h, device=dev())


def test_repeated_solves_with_poisoned_scratch_and_graph_cache():
    w = tdma_inputs.make_workload("cfg1_tiny", device=dev())
    x1 = torch.empty_like(w.d)
    x2 = torch.empty_like(w.d)
    with tdma.Plan(w.nx, w.ny, w.nz, w.P, 8, variant=tdma.TDMA_VARIANT_PIPELINED, nstreams=3) as plan:
        plan.solve(w.a, w.b, w.c, w.d, x1)
        torch.cuda.synchronize()
        for which in (tdma.TDMA_BUF_SA, tdma.TDMA_BUF_SC, tdma.TDMA_BUF_SD, tdma.TDMA_BUF_RA,
                      tdma.TDMA_BUF_RC, tdma.TDMA_BUF_RD, tdma.TDMA_BUF_Y):
            for slot in range(plan.get(tdma.TDMA_GET_DEPTH)):
                ptr, nbytes = plan.buffer(which, slot)
                _view(ptr, nbytes, (nbytes // 8,)).fill_(float("nan"))
        torch.cuda.synchronize()
        plan.solve(w.a, w.b, w.c, w.d, x2)          # same inputs, other x -> a second graph
        x1.fill_(float("nan"))
        plan.solve(w.a, w.b, w.c, w.d, x1)          # cached graph
        torch.cuda.synchronize()
        assert plan.get(tdma.TDMA_GET_GRAPH_BUILDS) == 2
    assert torch.equal(x1, x2)
    check_against_oracle(w.a, w.b, w.c, w.d, x1, True)


# ---------------------------------------------------------------------------------------------
# Degenerate and ragged cases
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("shape,P,batch", [
    ((7, 64, 100), 4, 3),      # nx not a multiple of 32 (pipelined) / of 8 handled below
    ((3, 32, 8), 16, 2),       # m = 2: partitions without interior rows
    ((1, 48, 64), 1, 0),       # P = 1 degenerates to a plain solve
    ((5, 6, 16), 3, 5),        # m = 2, tiny
    ((2, 96, 40), 2, 1),       # m = 48
    ((9, 30, 24), 5, 4),       # m = 6, nz % batch != 0
    ((1, 2, 8), 1, 0),         # ny = 2
])
def test_shapes(variant, shape, P, batch):
    nz, ny, nx = shape
    a, b, c, d = tdma_inputs.dominant_random(nx, ny, nz, 11, dev())
    try:
        x = gpu_solve(a, b, c, d, P, batch, **variant)
    except tdma.TdmaError as exc:
        if variant["variant"] == tdma.TDMA_VARIANT_FUSED and "fused variant unavailable" in str(exc):
            pytest.skip(str(exc))
        if variant["variant"] == tdma.TDMA_VARIANT_STAGED and "STAGED variant unavailable" in str(exc):
            pytest.skip(str(exc))       # shapes the TMA kernel cannot tile (30 rows: no power-of-two tree)
        raise
    check_against_oracle(a, b, c, d, x, True)


@pytest.mark.parametrize("shape,P", [((4, 16, 1), 4), ((1, 16, 37), 2), ((3, 1, 5), 1), ((2, 10, 3), 1)])
def test_odd_nx_pipelined(shape, P):
    nz, ny, nx = shape
    a, b, c, d = tdma_inputs.dominant_random(nx, ny, nz, 5, dev())
    x = gpu_solve(a, b, c, d, P, 0, variant=tdma.TDMA_VARIANT_PIPELINED)
    check_against_oracle(a, b, c, d, x, True)


@pytest.mark.parametrize("shape,P", [((4, 16, 1), 4), ((1, 16, 37), 2), ((2, 10, 3), 1), ((3, 64, 45), 4)])
def test_odd_nx_fused(shape, P):
    """Ragged x tail: lanes past nx compute a copy of the last line and store nothing."""
    nz, ny, nx = shape
    a, b, c, d = tdma_inputs.dominant_random(nx, ny, nz, 5, dev())
    guard = torch.full((nz * ny * nx + 64,), float("nan"), dtype=torch.float64, device=dev())
    x = guard[:nz * ny * nx].view(nz, ny, nx)
    gpu_solve(a, b, c, d, P, 0, variant=tdma.TDMA_VARIANT_FUSED, out=x)
    assert torch.isnan(guard[nz * ny * nx:]).all()
    check_against_oracle(a, b, c, d, x, True)


def test_fused_rejects_what_it_cannot_tile():
    with pytest.raises(tdma.TdmaError) as ei:     # P = 1 keeps the whole line in one CTA
        tdma.Plan(64, 4096, 2, 1, 0, variant=tdma.TDMA_VARIANT_FUSED, fused_impl=1)
    assert "fused variant unavailable" in str(ei.value)
    with pytest.raises(tdma.TdmaError):
        tdma.Plan(64, 64, 2, 4, 0, variant=tdma.TDMA_VARIANT_FUSED, fused_lines=64)
    with pytest.raises(tdma.TdmaError) as ei:     # TMA needs 16-byte global strides
        tdma.Plan(45, 64, 2, 4, 0, **TMA)
    assert "even nx" in str(ei.value)
    with pytest.raises(tdma.TdmaError):           # 48 = 3 * 16: no power-of-two tree
        tdma.Plan(64, 96, 2, 2, 0, fused_leaf_rows=16, **TMA)


# ---------------------------------------------------------------------------------------------
# TMA fused kernel: tilings (lines x cluster x leaf), ragged x tiles, alignment fallback
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cluster,lines,leaf", [
    (1, 16, 0), (1, 16, 2), (1, 8, 16), (1, 16, 4), (2, 16, 8), (2, 32, 4), (4, 16, 2), (4, 8, 16),
    (8, 16, 8), (8, 32, 4), (8, 8, 2), (16, 16, 4), (16, 32, 2),
])
def test_tma_fused_tilings(cluster, lines, leaf):
    w = tdma_inputs.make_workload("cfg1_tiny", device=dev())
    with tdma.Plan(w.nx, w.ny, w.nz, w.P, 0, fused_cluster=cluster, fused_lines=lines,
                   fused_leaf_rows=leaf, **TMA) as plan:
        assert plan.get(tdma.TDMA_GET_FUSED_IMPL) == 2
        assert plan.get(tdma.TDMA_GET_FUSED_CLUSTER) == cluster
        assert plan.get(tdma.TDMA_GET_FUSED_LINES) == lines
        if leaf:
            assert plan.get(tdma.TDMA_GET_FUSED_LEAF_ROWS) == leaf
        assert plan.get(tdma.TDMA_GET_FUSED_TOP_ROWS) == 2 * cluster
        x = torch.full_like(w.d, float("nan"))
        plan.solve(w.a, w.b, w.c, w.d, x)
        torch.cuda.synchronize()
    check_against_oracle(w.a, w.b, w.c, w.d, x, True)


@pytest.mark.parametrize("shape,P,cluster,lines", [
    ((3, 64, 46), 4, 2, 16),      # ragged last x tile (46 = 2*16 + 14): TMA zero-fills / clips
    ((2, 1024, 20), 16, 8, 16),   # cfg-3 line length, tile wider than the ragged remainder
    ((2, 2048, 8), 32, 8, 8),     # two TMA boxes per array (R = 256 rows, box 256) -> R > 256 with CL = 4
    ((2, 2048, 8), 32, 4, 8),
    ((1, 2, 8), 1, 1, 8),         # ny = 2
    ((3, 32, 8), 16, 2, 8),       # m = 2: partitions without interior rows
])
def test_tma_fused_shapes(shape, P, cluster, lines):
    nz, ny, nx = shape
    a, b, c, d = tdma_inputs.dominant_random(nx, ny, nz, 13, dev())
    guard = torch.full((nz * ny * nx + 64,), float("nan"), dtype=torch.float64, device=dev())
    x = guard[:nz * ny * nx].view(nz, ny, nx)
    gpu_solve(a, b, c, d, P, 0, out=x, fused_cluster=cluster, fused_lines=lines, **TMA)
    assert torch.isnan(guard[nz * ny * nx:]).all()
    check_against_oracle(a, b, c, d, x, True)


@pytest.mark.parametrize("axis", ["y", "z"])
@pytest.mark.parametrize("n,P,cluster", [(768, 16, (3, 6)), (384, 8, (3,)), (640, 16, (5,)), (1280, 16, (5,)), (1536, 16, (6,))])
def test_odd_clusters_for_3_2k_and_5_2k_lines(axis, n, P, cluster):
    """AUTO on 3 * 2^k / 5 * 2^k line lengths: clusters of 3, 5 or 6 CTAs with 16-row leaves (256 threads), no
    fill launch; many tiles per cluster, repeated solves with equal bits, parity on the first and last slices."""
    lanes, nsl = 96, 40
    shape = (nsl, n, lanes) if axis == "y" else (n, nsl, lanes)
    a, b, c, d = tdma_inputs.dominant_random(shape[2], shape[1], shape[0], 17, dev())
    xs = []
    with tdma.Plan(shape[2], shape[1], shape[0], P, 0, axis=tdma.TDMA_AXIS_Z if axis == "z" else tdma.TDMA_AXIS_Y) as plan:
        assert plan.get(tdma.TDMA_GET_VARIANT) == tdma.TDMA_VARIANT_FUSED
        assert plan.get(tdma.TDMA_GET_FUSED_CLUSTER) in cluster and plan.get(tdma.TDMA_GET_FUSED_LEAF_ROWS) == 16
        for _ in range(4):
            x = torch.full_like(d, float("nan"))
            plan.solve(a, b, c, d, x)
            xs.append(x)
        torch.cuda.synchronize()
        assert plan.get(tdma.TDMA_GET_FUSED_FILL) == 0
    assert all(torch.equal(xs[0], t) for t in xs[1:])
    an, bn, cn, dn, xn = to_np(a, b, c, d, xs[0])
    ref = oracle.solve_axis(an, bn, cn, dn, axis, False)
    ax = 1 if axis == "y" else 0
    err = (np.max(np.abs(xn - ref), axis=ax) / np.max(np.abs(ref), axis=ax)).max()
    assert np.isfinite(xn).all() and err <= TOL_E, err


def test_tma_fused_unaligned_pointers_fall_back():
    """Arrays that are only 8-byte aligned cannot be described by a tensor map: the plan routes
    the solve to the register-staged kernel instead of failing."""
    w = tdma_inputs.make_workload("cfg1_tiny", device=dev())
    n = w.d.numel()
    bufs = [torch.empty(n + 1, dtype=torch.float64, device=dev()) for _ in range(5)]
    views = [b[1:].view_as(w.d) for b in bufs]
    for v, t in zip(views, (w.a, w.b, w.c, w.d)):
        v.copy_(t)
    assert views[0].data_ptr() % 16 == 8
    x = gpu_solve(views[0], views[1], views[2], views[3], w.P, 0, out=views[4], variant=tdma.TDMA_VARIANT_FUSED)
    check_against_oracle(w.a, w.b, w.c, w.d, x, True)


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("mode", ["up500", "down500", "mixed", "tiny_pivots"])
def test_row_scaling_extremes(variant, mode):
    """Numerical edge of the reciprocal path (D2: Newton reciprocal valid for pivots with
    2^-1021 < |p| < 2^1021, tree rows carried un-normalised).  Scaling row j of a system by 2^e_j
    leaves x unchanged and is exact in fp64, so the scaled system must still match the reference
    on the same scaled arrays: all rows x 2^500, all x 2^-500, a different power per row in
    [-300, 300], and pivots near 2^-1000."""
    nz, ny, nx = 3, 512, 64
    a, b, c, d = tdma_inputs.dominant_random(nx, ny, nz, 77, dev())
    g = torch.Generator().manual_seed(5)
    if mode == "up500":
        e = torch.full((nz, ny, nx), 500.0, dtype=torch.float64)
    elif mode == "down500":
        e = torch.full((nz, ny, nx), -500.0, dtype=torch.float64)
    elif mode == "mixed":
        e = torch.randint(-300, 301, (nz, ny, nx), generator=g).to(torch.float64)
    else:
        e = torch.full((nz, ny, nx), -1001.0, dtype=torch.float64)          # b in [2, 5) -> pivots ~ 2^-1000
    sc = torch.pow(torch.tensor(2.0, dtype=torch.float64), e).to(dev())
    a, b, c, d = a * sc, b * sc, c * sc, d * sc
    x = gpu_solve(a, b, c, d, 16, 0, **variant)
    an, bn, cn, dn, xn = to_np(a, b, c, d, x)
    assert np.isfinite(xn).all()
    ref = oracle.solve_y(an, bn, cn, dn, "f64")
    assert oracle.normwise_error(xn, ref).max() <= TOL_E


@pytest.mark.parametrize("variant", VARIANTS)
def test_identity_and_diagonal(variant):
    for diag in (False, True):
        a, b, c, d = tdma_inputs.identity_system(32, 16, 3, 2, dev(), diagonal_only=diag)
        x = gpu_solve(a, b, c, d, 4, 2, **variant)
        # the kernels multiply by reciprocals (and the TMA kernel carries rows un-normalised):
        # a few ulp, not a correctly rounded quotient
        assert torch.allclose(x, d / b, rtol=1e-15, atol=0)


@pytest.mark.parametrize("variant", VARIANTS)
def test_corner_entries_are_ignored(variant):
    a, b, c, d = tdma_inputs.dominant_random(32, 24, 2, 3, dev())
    x0 = gpu_solve(a, b, c, d, 4, 0, **variant)
    a2, c2 = a.clone(), c.clone()
    a2[:, 0, :] = float("nan")
    c2[:, -1, :] = float("inf")
    x1 = gpu_solve(a2, b, c2, d, 4, 0, **variant)
    assert torch.equal(x0, x1)


@pytest.mark.parametrize("variant", VARIANTS)
def test_in_place_x_aliases_d(variant):
    w = tdma_inputs.make_workload("cfg1_tiny", device=dev())
    ref = gpu_solve(w.a, w.b, w.c, w.d, w.P, 16, **variant)
    buf = w.d.clone()
    gpu_solve(w.a, w.b, w.c, buf, w.P, 16, out=buf, **variant)
    assert torch.equal(buf, ref)


def test_inputs_are_not_written():
    w = tdma_inputs.make_workload("cfg1_tiny", device=dev())
    keep = [t.clone() for t in (w.a, w.b, w.c, w.d)]
    for variant in VARIANT_OPTS:
        gpu_solve(w.a, w.b, w.c, w.d, w.P, 8, **variant)
    for t, k in zip((w.a, w.b, w.c, w.d), keep):
        assert torch.equal(t, k)


def test_manufactured_solution_on_gpu():
    """P2 through the CUDA path: d = A x* (long double on the host), recover x*."""
    rng = np.random.default_rng(0)
    a, b, c, _ = tdma_inputs.dominant_random(64, 128, 3, 9, "cpu")
    xstar = rng.uniform(-1, 1, (3, 128, 64))
    d = oracle.apply_y(a.numpy(), b.numpy(), c.numpy(), xstar)
    dd = torch.from_numpy(d).to(dev())
    for variant in VARIANT_OPTS:
        x = gpu_solve(a.to(dev()), b.to(dev()), c.to(dev()), dd, 8, 2, **variant)
        assert oracle.normwise_error(x.cpu().numpy(), xstar).max() <= 1e-14


def test_toeplitz_closed_form_on_gpu():
    """P4 through the CUDA path: eigen-form of a=c=-alpha, b=1+2alpha."""
    n, alpha, nx = 512, 3.7, 32
    j = np.arange(1, n + 1)
    a = torch.full((1, n, nx), -alpha, dtype=torch.float64, device=dev())
    b = torch.full((1, n, nx), 1 + 2 * alpha, dtype=torch.float64, device=dev())
    d = np.zeros((1, n, nx))
    ref = np.zeros((1, n, nx))
    for q in range(1, nx + 1):
        mode = np.sin(np.pi * q * j / (n + 1))
        lam = 1 + 2 * alpha - 2 * alpha * np.cos(np.pi * q / (n + 1))
        d[0, :, q - 1] = mode
        ref[0, :, q - 1] = mode / lam
    dd = torch.from_numpy(d).to(dev())
    for variant in VARIANT_OPTS:
        x = gpu_solve(a, b, a, dd, 8, 0, **variant)
        assert oracle.normwise_error(x.cpu().numpy(), ref).max() <= (1 + 4 * alpha) * 2e-14


# ---------------------------------------------------------------------------------------------
# Stage level
# ---------------------------------------------------------------------------------------------
def test_stage_level_reduced_system_and_forward_rows():
    w = tdma_inputs.make_workload("cfg1_tiny", device=dev())
    P, m, Lb = w.P, w.ny // w.P, w.nx * w.nz
    an, bn, cn, dn = to_np(w.a, w.b, w.c, w.d)
    ref = oracle.solve_y(an, bn, cn, dn)                          # (nz, ny, nx)
    x = torch.empty_like(w.d)
    with tdma.Plan(w.nx, w.ny, w.nz, P, 0, variant=tdma.TDMA_VARIANT_PIPELINED) as plan:
        # stage-isolated entry point, in Alg. 1 order
        for st in (tdma.TDMA_STAGE_A, tdma.TDMA_STAGE_B, tdma.TDMA_STAGE_C):
            plan.stage(st, 0, w.a, w.b, w.c, w.d, x)
        torch.cuda.synchronize()
        bufs = {}
        for name, which, shape in [("RA", tdma.TDMA_BUF_RA, (2 * P, Lb)), ("RC", tdma.TDMA_BUF_RC, (2 * P, Lb)),
                                   ("RD", tdma.TDMA_BUF_RD, (2 * P, Lb)), ("Y", tdma.TDMA_BUF_Y, (2 * P, Lb)),
                                   ("SA", tdma.TDMA_BUF_SA, (w.nz, w.ny, w.nx)),
                                   ("SC", tdma.TDMA_BUF_SC, (w.nz, w.ny, w.nx)),
                                   ("SD", tdma.TDMA_BUF_SD, (w.nz, w.ny, w.nx))]:
            ptr, nbytes = plan.buffer(which, 0)
            bufs[name] = _view(ptr, nbytes, shape).clone().cpu().numpy()
        x_full = torch.empty_like(w.d)
        plan.solve(w.a, w.b, w.c, w.d, x_full)
        torch.cuda.synchronize()
    assert torch.equal(x, x_full)                                  # stage API == whole solve
    RA, RC, RD, Y = bufs["RA"], bufs["RC"], bufs["RD"], bufs["Y"]
    # P6: diagonal dominance of the reduced system, zero corners, Y = oracle x at partition ends
    assert (np.abs(RA) + np.abs(RC) < 1).all()
    assert (RA[0] == 0).all() and (RC[2 * P - 1] == 0).all()
    ref_lines = ref.transpose(1, 0, 2).reshape(w.ny, Lb)           # line index = i + nx*k
    for p in range(P):
        assert np.max(np.abs(Y[2 * p] - ref_lines[p * m])) <= 1e-14
        assert np.max(np.abs(Y[2 * p + 1] - ref_lines[p * m + m - 1])) <= 1e-14
        # reduced rows hold for the oracle solution
        xf, xl = ref_lines[p * m], ref_lines[p * m + m - 1]
        xprev = ref_lines[p * m - 1] if p > 0 else 0 * xf
        xnext = ref_lines[p * m + m] if p < P - 1 else 0 * xf
        assert np.max(np.abs(RA[2 * p] * xprev + xf + RC[2 * p] * xl - RD[2 * p])) <= 1e-14
        assert np.max(np.abs(RA[2 * p + 1] * xf + xl + RC[2 * p + 1] * xnext - RD[2 * p + 1])) <= 1e-14
    # P5 (forward-form rows): a'_r x_0 + x_r + c'_r x_{r+1} = d'_r for interior rows
    SA, SC, SD = bufs["SA"], bufs["SC"], bufs["SD"]
    for p in range(P):
        x0 = ref[:, p * m, :]
        for r in range(1, m - 1):
            j = p * m + r
            lhs = SA[:, j, :] * x0 + ref[:, j, :] + SC[:, j, :] * ref[:, j + 1, :]
            assert np.max(np.abs(lhs - SD[:, j, :])) <= 1e-14


@pytest.mark.parametrize("P,want_pe", [(4, 4), (16, 16), (32, 16)])
def test_staged_stage_level_reduced_system(P, want_pe):
    """STAGED (TMA-staged stage A / C, nothing spilled): the reduced rows stage A leaves in HBM hold
    for the oracle solution, stage B's Y equals the oracle at the ends of the exchanged nodes, and
    the stage-isolated calls reproduce the whole solve bit for bit.  256 rows: 16 leaves of 16
    rows; P = 4 exchanges the nodes of one 4-ary level (64 rows = the paper's partition), P = 16 the
    leaves, P = 32 (8-row partitions, shorter than a leaf) the leaves as well (D1)."""
    nx, ny, nz = 96, 256, 5
    a, b, c, d = tdma_inputs.dominant_random(nx, ny, nz, 61, dev())
    an, bn, cn, dn = to_np(a, b, c, d)
    ref = oracle.solve_y(an, bn, cn, dn)
    x = torch.full_like(d, float("nan"))
    with tdma.Plan(nx, ny, nz, P, 0, variant=tdma.TDMA_VARIANT_STAGED) as plan:
        pe = plan.get(tdma.TDMA_GET_REDUCED_PARTITIONS)
        assert pe == want_pe
        for st in (tdma.TDMA_STAGE_A, tdma.TDMA_STAGE_B, tdma.TDMA_STAGE_C):
            plan.stage(st, 0, a, b, c, d, x)
        torch.cuda.synchronize()
        Lb, m = nx * nz, ny // pe
        bufs = {}
        for name, which in (("RA", tdma.TDMA_BUF_RA), ("RC", tdma.TDMA_BUF_RC), ("RD", tdma.TDMA_BUF_RD), ("Y", tdma.TDMA_BUF_Y)):
            ptr, nbytes = plan.buffer(which, 0)
            bufs[name] = _view(ptr, nbytes, (2 * pe, Lb)).clone().cpu().numpy()
        with pytest.raises(tdma.TdmaError):
            plan.buffer(tdma.TDMA_BUF_SA, 0)                       # there is no scratch ring
        assert plan.workspace_bytes == 3 * 5 * 2 * pe * Lb * 8     # reduced buffers only
        x_full = torch.empty_like(d)
        plan.solve(a, b, c, d, x_full)
        torch.cuda.synchronize()
    assert torch.equal(x, x_full)
    check_against_oracle(a, b, c, d, x, True)
    RA, RC, RD, Y = bufs["RA"], bufs["RC"], bufs["RD"], bufs["Y"]
    assert (RA[0] == 0).all() and (RC[2 * pe - 1] == 0).all()
    ref_lines = ref.transpose(1, 0, 2).reshape(ny, Lb)
    for p in range(pe):
        xf, xl = ref_lines[p * m], ref_lines[p * m + m - 1]
        assert np.max(np.abs(Y[2 * p] - xf)) <= 1e-13 and np.max(np.abs(Y[2 * p + 1] - xl)) <= 1e-13
        xprev = ref_lines[p * m - 1] if p > 0 else 0 * xf
        xnext = ref_lines[p * m + m] if p < pe - 1 else 0 * xf
        assert np.max(np.abs(RA[2 * p] * xprev + xf + RC[2 * p] * xl - RD[2 * p])) <= 1e-13
        assert np.max(np.abs(RA[2 * p + 1] * xf + xl + RC[2 * p + 1] * xnext - RD[2 * p + 1])) <= 1e-13


def test_staged_schedule_invariance():
    """STAGED: x does not depend on batching, stream count or graph capture (G13)."""
    w = tdma_inputs.make_workload("cfg1_tiny", device=dev())
    base = gpu_solve(w.a, w.b, w.c, w.d, w.P, 0, variant=tdma.TDMA_VARIANT_STAGED)
    for batch, opts in [(1, {}), (7, dict(nstreams=3)), (16, dict(nstreams=1)), (24, dict(use_graph=-1)), (5, dict(nstreams=4))]:
        x = gpu_solve(w.a, w.b, w.c, w.d, w.P, batch, variant=tdma.TDMA_VARIANT_STAGED, **opts)
        assert torch.equal(x, base), (batch, opts)


# ---------------------------------------------------------------------------------------------
# PDD variant of stage B
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", [tdma.TDMA_VARIANT_PIPELINED, tdma.TDMA_VARIANT_STAGED], ids=["pipelined", "staged"])
@pytest.mark.parametrize("kind", ["random", "adi_0.3", "adi_8"])
def test_pdd_stage_b_matches_the_pdd_reference(variant, kind):
    """options.pdd: stage B solves the 2 x 2 interface systems of Sun's PDD.  An approximation, so
    the reference is oracle.solve_y_pdd for the same partition count (element-wise parity at 1e-11:
    both sides drop the same entries), and the distance to the EXACT solve is checked against the
    size of what was dropped (alpha = 8: r = 0.70, 64-row partitions -> ~1e-10 relative)."""
    nx, ny, nz, P = 64, 256, 4, 4
    if kind == "random":
        a, b, c, d = tdma_inputs.dominant_random(nx, ny, nz, 71, dev())
    else:
        a, b, c, d, _ = tdma_inputs.adi_toeplitz(nx, ny, nz, 72, dev(), alpha=float(kind.split("_")[1]))
    x = torch.full_like(d, float("nan"))
    with tdma.Plan(nx, ny, nz, P, 2, variant=variant, pdd=1) as plan:
        pe = plan.get(tdma.TDMA_GET_REDUCED_PARTITIONS)
        plan.solve(a, b, c, d, x)
        torch.cuda.synchronize()
    an, bn, cn, dn, xn = to_np(a, b, c, d, x)
    ref = oracle.solve_y_pdd(an, bn, cn, dn, pe)
    assert oracle.normwise_error(xn, ref).max() <= TOL_E
    exact = oracle.solve_y(an, bn, cn, dn)
    gap, own = oracle.normwise_error(xn, exact).max(), oracle.normwise_error(ref, exact).max()
    assert gap <= 2 * own + 1e-13                      # the GPU is as far from exact as the reference is
    if kind == "adi_0.3":
        assert gap <= 1e-13                            # r = 0.22: r^63 is far below rounding
    with pytest.raises(tdma.TdmaError):
        tdma.Plan(nx, ny, nz, P, 0, variant=tdma.TDMA_VARIANT_FUSED, pdd=1)


# ---------------------------------------------------------------------------------------------
# Host-buffer entry point
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", VARIANTS)
def test_solve_host_matches_device_solve(variant):
    w = tdma_inputs.make_workload("cfg2_poisson", device="cpu", nx=64, nz=40)
    host = [t.pin_memory() for t in (w.a, w.b, w.c, w.d)]
    xh = torch.empty_like(w.d).pin_memory()
    with tdma.Plan(w.nx, w.ny, w.nz, w.P, 4, **variant) as plan:
        plan.solve_host(*host, xh)
        xd = torch.empty_like(w.d, device=dev())
        plan.solve(*[t.to(dev()) for t in host], xd)
        torch.cuda.synchronize()
    assert torch.equal(xh, xd.cpu())
    check_against_oracle(w.a, w.b, w.c, w.d, xh, False)


def test_solve_on_non_default_stream_orders_with_later_work():
    w = tdma_inputs.make_workload("cfg1_tiny", device=dev())
    ref = gpu_solve(w.a, w.b, w.c, w.d, w.P, 8, variant=tdma.TDMA_VARIANT_PIPELINED)
    s = torch.cuda.Stream()
    x = torch.zeros_like(w.d)
    y = torch.zeros_like(w.d)
    with tdma.Plan(w.nx, w.ny, w.nz, w.P, 8, variant=tdma.TDMA_VARIANT_PIPELINED, use_graph=-1) as plan:
        s.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(s):
            plan.solve(w.a, w.b, w.c, w.d, x, stream=s)
            y.copy_(x)                       # later work on the same stream must see x
        s.synchronize()
    assert torch.equal(y, ref)


def test_pipeline_timeline_records_alg2_order():
    """options.timeline: every stage launch of the last solve with start <= end, per batch
    A before B before C (the event dependencies of Alg. 2), results unchanged."""
    w = tdma_inputs.make_workload("cfg1_tiny", device=dev())
    ref = gpu_solve(w.a, w.b, w.c, w.d, w.P, 8, variant=tdma.TDMA_VARIANT_PIPELINED)
    x = torch.empty_like(w.d)
    with tdma.Plan(w.nx, w.ny, w.nz, w.P, 8, variant=tdma.TDMA_VARIANT_PIPELINED, nstreams=3, timeline=1) as plan:
        plan.solve(w.a, w.b, w.c, w.d, x)
        recs = plan.timeline()
    assert torch.equal(x, ref)
    nb = w.nz // 8
    assert len(recs) == 3 * nb
    by = {(s, b): (t0, t1) for s, b, t0, t1 in recs}
    for b in range(nb):
        A, B, C = by[(tdma.TDMA_STAGE_A, b)], by[(tdma.TDMA_STAGE_B, b)], by[(tdma.TDMA_STAGE_C, b)]
        assert A[0] <= A[1] and B[0] <= B[1] and C[0] <= C[1]
        assert A[1] <= B[1] + 1e-3 and B[1] <= C[1] + 1e-3


def test_fill_launch_changes_x_only_within_rounding():
    """G13 scoped: the fill launch solves its slices with another tiling (clusters of 2,
    8 lines), so the BITS of x in the fill range depend on where that range starts; the values
    agree with the no-fill solve and with the oracle to the tolerance."""
    w = tdma_inputs.make_workload("cfg3_weak", device=dev(), nz=48)
    with tdma.Plan(w.nx, w.ny, w.nz, w.P, 0, variant=tdma.TDMA_VARIANT_FUSED) as plan:
        x_auto = torch.full_like(w.d, float("nan"))
        plan.solve(w.a, w.b, w.c, w.d, x_auto)
        torch.cuda.synchronize()
        fill = plan.get(tdma.TDMA_GET_FUSED_FILL)
    x_off = gpu_solve(w.a, w.b, w.c, w.d, w.P, 0, variant=tdma.TDMA_VARIANT_FUSED, fused_fill=-1)
    x_big = gpu_solve(w.a, w.b, w.c, w.d, w.P, 0, variant=tdma.TDMA_VARIANT_FUSED, fused_fill=500)
    if fill > 0:
        assert torch.equal(x_auto[:w.nz - fill], x_off[:w.nz - fill])      # main range: same tiling, same bits
    for x in (x_auto, x_off, x_big):
        check_against_oracle(w.a, w.b, w.c, w.d, x, False)
    E = oracle.normwise_error(x_auto.cpu().numpy(), x_off.cpu().numpy())
    assert E.max() <= TOL_E


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("chunk", [3, 16])
def test_solve_host_streams_several_chunks(variant, chunk):
    """tdma_solve_host with >= 3 chunks and a ragged last one (40 = 3*13 + 1 / 16+16+8): the
    double-buffered staging ring (slot reuse waits on solve + D2H of chunk q-2) and the second
    graph of the ragged chunk are exercised; PIPELINED rounds the chunk to whole batches, so its
    bits equal tdma_solve's."""
    w = tdma_inputs.make_workload("cfg2_poisson", device="cpu", nx=64, nz=40)
    host = [t.pin_memory() for t in (w.a, w.b, w.c, w.d)]
    xh = torch.full_like(w.d, float("nan")).pin_memory()
    batch = 4
    with tdma.Plan(w.nx, w.ny, w.nz, w.P, batch, host_chunk=chunk, **variant) as plan:
        plan.solve_host(*host, xh)
        xh2 = torch.full_like(w.d, float("nan")).pin_memory()
        plan.solve_host(*host, xh2)                  # staging buffers and graphs reused
        xd = torch.empty_like(w.d, device=dev())
        plan.solve(*[t.to(dev()) for t in host], xd)
        torch.cuda.synchronize()
    assert torch.equal(xh, xh2)
    assert torch.equal(xh, xd.cpu())                 # no fill launch at this size: same tiling per slice
    check_against_oracle(w.a, w.b, w.c, w.d, xh, False)
