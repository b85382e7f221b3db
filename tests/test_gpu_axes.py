"""SURVEY 8(f) f1 (BASELINE cfg 4, ADI sweeps): z sweeps and cyclic lines through the C ABI against
the oracle (oracle.solve_axis), element by element: x, y and z sweeps, plain and cyclic lines."""
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


def solve(a, b, c, d, P, batch, **opts):
    nz, ny, nx = a.shape
    x = torch.full_like(d, float("nan"))
    with tdma.Plan(nx, ny, nz, P, batch, **opts) as plan:
        plan.solve(a, b, c, d, x)
        torch.cuda.synchronize()
    return x


def check(a, b, c, d, x, axis, periodic):
    an, bn, cn, dn, xn = [t.cpu().numpy() for t in (a, b, c, d, x)]
    assert np.isfinite(xn).all()
    ref = oracle.solve_axis(an, bn, cn, dn, axis, periodic)
    ax = {"y": 1, "z": 0, "x": 2}[axis]
    err = np.max(np.abs(xn - ref), axis=ax) / np.max(np.abs(ref), axis=ax)
    assert err.max() <= TOL_E, err.max()


@pytest.mark.parametrize("opts", [dict(variant=tdma.TDMA_VARIANT_PIPELINED), dict(variant=tdma.TDMA_VARIANT_FUSED),
                                  dict(variant=tdma.TDMA_VARIANT_STAGED)], ids=["pipelined", "fused_tma", "staged"])
@pytest.mark.parametrize("shape,P,batch", [((64, 48, 32), 4, 0), ((256, 20, 64), 8, 7), ((32, 3, 46), 16, 2),
                                           ((512, 6, 128), 8, 4)])
def test_z_sweep(opts, shape, P, batch):
    nz, ny, nx = shape
    a, b, c, d = tdma_inputs.dominant_random(nx, ny, nz, 21, dev())
    x = solve(a, b, c, d, P, batch, axis=tdma.TDMA_AXIS_Z, **opts)
    check(a, b, c, d, x, "z", False)


@pytest.mark.parametrize("axis", ["y", "z"])
@pytest.mark.parametrize("n,P,cluster", [(64, 4, 0), (64, 4, 1), (256, 8, 4), (512, 8, 0), (1024, 16, 0), (8, 2, 2)])
def test_cyclic_lines(axis, n, P, cluster):
    other, nx = 6, 64
    shape = (other, n, nx) if axis == "y" else (n, other, nx)
    a, b, c, d = tdma_inputs.dominant_random(shape[2], shape[1], shape[0], 31, dev())
    x = solve(a, b, c, d, P, 0, variant=tdma.TDMA_VARIANT_FUSED, periodic=1, fused_cluster=cluster,
              axis=tdma.TDMA_AXIS_Z if axis == "z" else tdma.TDMA_AXIS_Y)
    check(a, b, c, d, x, axis, True)


def test_cfg4_adi_y_then_z_periodic_circulant_closed_form():
    """cfg 4 coefficients (a = c = -alpha, b = 1 + 2 alpha): Dirichlet y sweep followed by a
    periodic z sweep, the second one checked against the circulant closed form as well."""
    w = tdma_inputs.make_workload("cfg4_adi_y", device=dev(), nx=64, ny=128, nz=256, P=8)
    alpha = w.meta["alpha"]
    x1 = solve(w.a, w.b, w.c, w.d, w.P, 32, variant=tdma.TDMA_VARIANT_FUSED)
    check(w.a, w.b, w.c, w.d, x1, "y", False)
    x2 = solve(w.a, w.b, w.c, x1, w.P, 0, variant=tdma.TDMA_VARIANT_FUSED, axis=tdma.TDMA_AXIS_Z, periodic=1)
    check(w.a, w.b, w.c, x1, x2, "z", True)
    lam = 1 + 2 * alpha - 2 * alpha * np.cos(2 * np.pi * np.arange(w.nz) / w.nz)
    ref = np.fft.ifft(np.fft.fft(x1.cpu().numpy(), axis=0) / lam[:, None, None], axis=0).real
    assert np.max(np.abs(x2.cpu().numpy() - ref)) <= (1 + 4 * alpha) * 1e-13 * np.max(np.abs(ref))


@pytest.mark.parametrize("periodic", [0, 1])
@pytest.mark.parametrize("shape,P,cluster", [((3, 40, 64), 4, 0), ((2, 16, 256), 8, 1), ((4, 37, 512), 8, 2),
                                             ((2, 50, 1024), 16, 4), ((1, 20, 2048), 16, 8), ((5, 7, 16), 1, 1)])
def test_x_sweep(periodic, shape, P, cluster):
    """Lines along the contiguous axis: swizzled TMA boxes in, staging tile + TMA store out;
    ny not a multiple of the 16-line tile exercises the zero-fill / clipping."""
    nz, ny, nx = shape
    a, b, c, d = tdma_inputs.dominant_random(nx, ny, nz, 41, dev())
    guard = torch.full((nz * ny * nx + 64,), float("nan"), dtype=torch.float64, device=dev())
    x = guard[:nz * ny * nx].view(nz, ny, nx)
    with tdma.Plan(nx, ny, nz, P, 0, variant=tdma.TDMA_VARIANT_FUSED, axis=tdma.TDMA_AXIS_X, periodic=periodic,
                   fused_cluster=cluster) as plan:
        plan.solve(a, b, c, d, x)
        torch.cuda.synchronize()
    assert torch.isnan(guard[nz * ny * nx:]).all()
    check(a, b, c, d, x, "x", bool(periodic))


def test_cfg4_adi_three_sweeps():
    """BASELINE cfg 4 at reduced size: successive solves along x (periodic), y (Dirichlet) and z
    (periodic) with a = c = -alpha, b = 1 + 2 alpha; each against the oracle."""
    w = tdma_inputs.make_workload("cfg4_adi_y", device=dev(), nx=256, ny=128, nz=64, P=8)
    F = tdma.TDMA_VARIANT_FUSED
    x1 = solve(w.a, w.b, w.c, w.d, w.P, 0, variant=F, axis=tdma.TDMA_AXIS_X, periodic=1)
    check(w.a, w.b, w.c, w.d, x1, "x", True)
    x2 = solve(w.a, w.b, w.c, x1, w.P, 0, variant=F)
    check(w.a, w.b, w.c, x1, x2, "y", False)
    x3 = solve(w.a, w.b, w.c, x2, w.P, 0, variant=F, axis=tdma.TDMA_AXIS_Z, periodic=1)
    check(w.a, w.b, w.c, x2, x3, "z", True)


def test_cfg4_adi_full_size_three_sweeps_sampled():
    """BASELINE cfg 4 at FULL size (512^3, P = 8) in the plans `bench.py --adi` times (FUSED, auto
    tiling, batch = 0): x periodic -> y Dirichlet -> z periodic, every
    sweep against oracle.solve_axis on sampled z-slices (x, y sweeps) / y-planes (z sweep),
    including the slices a fill launch wrote."""
    w = tdma_inputs.make_workload("cfg4_adi_y", device=dev())
    F = tdma.TDMA_VARIANT_FUSED
    src = w.d
    for axis, name, periodic in ((tdma.TDMA_AXIS_X, "x", 1), (tdma.TDMA_AXIS_Y, "y", 0), (tdma.TDMA_AXIS_Z, "z", 1)):
        dst = torch.full_like(w.d, float("nan"))
        with tdma.Plan(w.nx, w.ny, w.nz, w.P, 0, variant=F, axis=axis, periodic=periodic) as plan:
            plan.solve(w.a, w.b, w.c, src, dst)
            torch.cuda.synchronize()
            fill = plan.get(tdma.TDMA_GET_FUSED_FILL)
        assert bool(torch.isfinite(dst).all())
        nsl = w.ny if name == "z" else w.nz
        picks = {0, 1, nsl // 2 + 1, nsl - 1}
        if fill > 0:
            picks |= {nsl - fill, nsl - fill - 1}
        for q in sorted(picks):
            sl = (slice(None), slice(q, q + 1)) if name == "z" else (slice(q, q + 1),)
            check(w.a[sl], w.b[sl], w.c[sl], src[sl], dst[sl], name, bool(periodic))
        src = dst


@pytest.mark.parametrize("axis", ["y", "z"])
@pytest.mark.parametrize("n,P,lanes,other,batch,nstreams", [
    (113, 1, 31, 5, 0, 2), (12, 6, 43, 27, 26, 2), (177, 59, 1022, 3, 2, 3), (64, 4, 64, 6, 0, 1), (3, 1, 7, 4, 1, 2),
    (768, 16, 77, 4, 3, 2), (2048, 256, 31, 2, 0, 2), (1024, 16, 256, 3, 2, 4)])
def test_cyclic_lines_on_the_stage_pipeline(axis, n, P, lanes, other, batch, nstreams):
    """Cyclic lines in the PIPELINED variant: stage A keeps a_0 and c_{n-1}, stage B solves the cyclic
    2P-row reduced system, stage C is unchanged.  Any nx (odd included) and any line length, i.e. the
    shapes the TMA kernel cannot tile; P = 1 (a two-row reduced system), ragged last batch, 1-4 streams."""
    shape = (other, n, lanes) if axis == "y" else (n, other, lanes)
    a, b, c, d = tdma_inputs.dominant_random(shape[2], shape[1], shape[0], 71, dev())
    x = solve(a, b, c, d, P, batch, variant=tdma.TDMA_VARIANT_PIPELINED, periodic=1, nstreams=nstreams,
              axis=tdma.TDMA_AXIS_Z if axis == "z" else tdma.TDMA_AXIS_Y)
    check(a, b, c, d, x, axis, True)


@pytest.mark.parametrize("periodic", [0, 1])
@pytest.mark.parametrize("nx,cluster", [(48, 3), (96, 3), (384, 3), (768, 3), (1536, 6), (768, 6), (80, 5), (320, 5), (640, 5),
                                        (1280, 5)])
def test_x_sweeps_of_3_2k_cells(nx, cluster, periodic):
    """x sweeps whose lines hold 3 * 2^k or 5 * 2^k cells: the leaves are whole 128-byte rows of 16 x, so the odd
    factor goes into the cluster (3, 6 or 5 CTAs per line tile) instead of the leaf.  General form and shared form (per-line
    shifts and uniform matrix), repeated solves with equal bits."""
    nz, ny = 3, 37
    a, b, c, d = tdma_inputs.dominant_random(nx, ny, nz, 45, dev())
    xs = []
    with tdma.Plan(nx, ny, nz, 1, 0, axis=tdma.TDMA_AXIS_X, periodic=periodic, fused_cluster=cluster if nx == 768 else 0) as plan:
        assert plan.get(tdma.TDMA_GET_VARIANT) == tdma.TDMA_VARIANT_FUSED
        assert plan.get(tdma.TDMA_GET_FUSED_CLUSTER) == cluster
        for _ in range(4):
            x = torch.full_like(d, float("nan"))
            plan.solve(a, b, c, d, x)
            xs.append(x)
        torch.cuda.synchronize()
    check(a, b, c, d, xs[0], "x", bool(periodic))
    assert all(torch.equal(xs[0], t) for t in xs[1:])
    g = torch.Generator().manual_seed(nx)
    u = lambda k, lo, hi: lo + (hi - lo) * torch.rand(k, dtype=torch.float64, generator=g)
    a1, c1, b01, sy, sz = u(nx, -1, 1), u(nx, -1, 1), u(nx, 2.5, 3.5), -u(ny, 0, 2), -u(nz, 0, 2)
    dd = torch.randn((nz, ny, nx), dtype=torch.float64, generator=g)
    for uniform in (False, True):
        x = torch.full_like(dd, float("nan")).to(dev())
        with tdma.Plan(nx, ny, nz, 1, 0, axis=tdma.TDMA_AXIS_X, periodic=periodic) as plan:
            plan.solve_shared(*[t.to(dev()) for t in (a1, b01, c1)], None if uniform else sy.to(dev()),
                              None if uniform else sz.to(dev()), dd.to(dev()), x)
            torch.cuda.synchronize()
            assert plan.get(tdma.TDMA_GET_SHARED_LINE_KERNEL) == 0 and plan.get(tdma.TDMA_GET_SHARED_CLUSTER) in (3, 6, 5)
        A = a1.view(1, 1, nx).expand(nz, ny, nx).contiguous()
        C = c1.view(1, 1, nx).expand(nz, ny, nx).contiguous()
        B = (b01.view(1, 1, nx) - (0 if uniform else sy.view(1, ny, 1) + sz.view(nz, 1, 1))).expand(nz, ny, nx).contiguous()
        check(A, B, C, dd, x, "x", bool(periodic))


@pytest.mark.parametrize("periodic", [0, 1])
@pytest.mark.parametrize("shape,P,batch", [((3, 40, 115), 5, 2), ((2, 16, 49), 7, 0), ((4, 37, 18), 1, 3), ((1, 5, 3), 1, 0),
                                           ((5, 33, 176), 2, 4), ((2, 70, 1024), 16, 1)])
def test_x_sweep_on_the_stage_pipeline(periodic, shape, P, batch):
    """Lines along the contiguous axis in the PIPELINED variant (one thread per (line, partition), strided
    accesses): the fallback for line lengths the TMA kernel cannot tile -- odd nx, nx not a multiple of 16 --
    and what AUTO resolves to for them."""
    nz, ny, nx = shape
    a, b, c, d = tdma_inputs.dominant_random(nx, ny, nz, 43, dev())
    x = solve(a, b, c, d, P, batch, variant=tdma.TDMA_VARIANT_PIPELINED, axis=tdma.TDMA_AXIS_X, periodic=periodic)
    check(a, b, c, d, x, "x", bool(periodic))
    if nx % 16:
        with tdma.Plan(nx, ny, nz, P, batch, axis=tdma.TDMA_AXIS_X, periodic=periodic) as plan:
            assert plan.get(tdma.TDMA_GET_VARIANT) == tdma.TDMA_VARIANT_PIPELINED


@pytest.mark.parametrize("axis", ["y", "z"])
@pytest.mark.parametrize("n,P,batch", [(64, 4, 0), (256, 8, 2), (1024, 16, 3), (768, 16, 0), (32, 16, 1)])
def test_cyclic_lines_staged(axis, n, P, batch):
    """Cyclic lines in the STAGED variant: the TMA-staged stage A / C kernels keep a_0 and c_{n-1}, stage B
    is the cyclic reduced solve."""
    other, nx = 5, 96
    shape = (other, n, nx) if axis == "y" else (n, other, nx)
    a, b, c, d = tdma_inputs.dominant_random(shape[2], shape[1], shape[0], 75, dev())
    x = solve(a, b, c, d, P, batch, variant=tdma.TDMA_VARIANT_STAGED, periodic=1,
              axis=tdma.TDMA_AXIS_Z if axis == "z" else tdma.TDMA_AXIS_Y)
    check(a, b, c, d, x, axis, True)


def test_cyclic_lines_auto_falls_back_to_the_stage_pipeline():
    """AUTO: cyclic lines go to the fused TMA kernel when the shape tiles, else to PIPELINED; both against
    the oracle, and against each other to rounding on a shape both can run."""
    a, b, c, d = tdma_inputs.dominant_random(45, 30, 8, 73, dev())             # odd nx
    x = torch.full_like(d, float("nan"))
    with tdma.Plan(45, 30, 8, 5, 2, periodic=1) as plan:
        assert plan.get(tdma.TDMA_GET_VARIANT) == tdma.TDMA_VARIANT_PIPELINED
        plan.solve(a, b, c, d, x)
        torch.cuda.synchronize()
    check(a, b, c, d, x, "y", True)
    a, b, c, d = tdma_inputs.dominant_random(64, 256, 6, 74, dev())
    with tdma.Plan(64, 256, 6, 8, 0, periodic=1) as plan:
        assert plan.get(tdma.TDMA_GET_VARIANT) == tdma.TDMA_VARIANT_FUSED
    xf = solve(a, b, c, d, 8, 0, variant=tdma.TDMA_VARIANT_FUSED, periodic=1)
    xp = solve(a, b, c, d, 8, 2, variant=tdma.TDMA_VARIANT_PIPELINED, periodic=1)
    check(a, b, c, d, xp, "y", True)
    assert float((xf - xp).abs().max() / xf.abs().max()) <= 1e-13


def test_cyclic_pipelined_circulant_closed_form():
    """cfg 4's periodic z sweep (a = c = -alpha, b = 1 + 2 alpha) through the PIPELINED variant against
    the circulant closed form x = IFFT(FFT(d) / lambda), lambda_q = 1 + 2 alpha - 2 alpha cos(2 pi q / n)."""
    w = tdma_inputs.make_workload("cfg4_adi_y", device=dev(), nx=48, ny=20, nz=200, P=8)
    alpha = w.meta["alpha"]
    x = solve(w.a, w.b, w.c, w.d, w.P, 7, variant=tdma.TDMA_VARIANT_PIPELINED, axis=tdma.TDMA_AXIS_Z, periodic=1)
    lam = 1 + 2 * alpha - 2 * alpha * np.cos(2 * np.pi * np.arange(w.nz) / w.nz)
    ref = np.fft.ifft(np.fft.fft(w.d.cpu().numpy(), axis=0) / lam[:, None, None], axis=0).real
    assert np.max(np.abs(x.cpu().numpy() - ref)) <= (1 + 4 * alpha) * 1e-13 * np.max(np.abs(ref))


def test_unsupported_combinations_fail_loudly():
    with pytest.raises(tdma.TdmaError):            # cyclic lines: not in the register-staged fused kernel
        tdma.Plan(32, 32, 32, 4, 0, variant=tdma.TDMA_VARIANT_FUSED, fused_impl=1, periodic=1)
    with pytest.raises(tdma.TdmaError):
        tdma.Plan(32, 32, 32, 4, 0, variant=tdma.TDMA_VARIANT_PIPELINED, periodic=1, pdd=1)
    with pytest.raises(tdma.TdmaError):
        tdma.Plan(32, 32, 32, 4, 0, variant=tdma.TDMA_VARIANT_FUSED, fused_impl=1, axis=tdma.TDMA_AXIS_Z)
    with pytest.raises(tdma.TdmaError):            # x sweeps: FUSED (TMA kernel) or PIPELINED
        tdma.Plan(32, 32, 32, 2, 0, variant=tdma.TDMA_VARIANT_STAGED, axis=tdma.TDMA_AXIS_X)
    with pytest.raises(tdma.TdmaError):            # x sweeps: 16-row leaves must tile the partitions
        tdma.Plan(24, 32, 32, 1, 0, variant=tdma.TDMA_VARIANT_FUSED, axis=tdma.TDMA_AXIS_X)
    with pytest.raises(tdma.TdmaError):
        tdma.Plan(32, 32, 32, 4, 0, axis=3)
    with pytest.raises(tdma.TdmaError):            # P must divide the line length (nz for a z sweep)
        tdma.Plan(32, 64, 30, 4, 0, axis=tdma.TDMA_AXIS_Z)


@pytest.mark.parametrize("shape,opts", [
    ((24, 1024, 1024), dict()), ((24, 1024, 1024), dict(fused_cluster=8)),
    ((24, 1024, 1024), dict(fused_cluster=2, fused_lines=8)),
    ((1024, 24, 1024), dict(axis=tdma.TDMA_AXIS_Z, periodic=1)), ((24, 512, 1024), dict(axis=tdma.TDMA_AXIS_X))],
    ids=["y_cl4_fill", "y_cl8", "y_cl2_tx8", "z_periodic", "x"])
def test_fused_tma_is_bitwise_reproducible(shape, opts):
    """The persistent kernel hands data between threads, CTAs (DSMEM inboxes double-buffered by
    tile parity) and launches (fill launch) with very few barriers; compute-sanitizer is closed on
    this pool, so races are hunted the blunt way: many tiles per cluster, repeated solves, every
    repeat must give the same bits (and a slab of the first one is checked against the oracle)."""
    nz, ny, nx = shape
    a, b, c, d = tdma_inputs.dominant_random(nx, ny, nz, 51, dev())
    xs = []
    with tdma.Plan(nx, ny, nz, 16, 0, variant=tdma.TDMA_VARIANT_FUSED, **opts) as plan:
        for rep in range(8):
            x = torch.full_like(d, float("nan"))
            plan.solve(a, b, c, d, x)
            xs.append(x)
        torch.cuda.synchronize()
        fill = plan.get(tdma.TDMA_GET_FUSED_FILL)
    for x in xs[1:]:
        assert torch.equal(x, xs[0])
    axis = {0: "y", 1: "x", 2: "z"}[opts.get("axis", 0)]
    nsl = nz if axis != "z" else ny                  # slices of the plan (z for x / y sweeps, y for z sweeps)
    ranges = [(0, 2)] + ([(nsl - fill, nsl)] if fill > 0 else [(nsl - 2, nsl)])   # + what the fill launch wrote
    for lo, hi in ranges:
        sl = (slice(lo, hi),) if axis != "z" else (slice(None), slice(lo, hi))
        check(a[sl], b[sl], c[sl], d[sl], xs[0][sl], axis, bool(opts.get("periodic", 0)))


def test_auto_variant_and_host_buffers_on_x_sweep():
    """tdma_plan_create (variant AUTO) resolves to FUSED when the shape tiles and to PIPELINED when
    it does not; tdma_solve_host works for x sweeps (z-chunks are contiguous)."""
    with tdma.Plan(64, 64, 8, 4, 2) as plan:
        assert plan.get(tdma.TDMA_GET_VARIANT) == tdma.TDMA_VARIANT_FUSED
        assert plan.get(tdma.TDMA_GET_NB) == 1          # batch is a hint for the stage pipelines only
    with tdma.Plan(45, 30, 8, 5, 2) as plan:            # odd nx, m = 6: no power-of-two tree
        assert plan.get(tdma.TDMA_GET_VARIANT) == tdma.TDMA_VARIANT_PIPELINED
        assert plan.get(tdma.TDMA_GET_NB) == 4
    a, b, c, d = tdma_inputs.dominant_random(128, 24, 6, 61, "cpu")
    host = [t.pin_memory() for t in (a, b, c, d)]
    xh = torch.empty_like(d).pin_memory()
    with tdma.Plan(128, 24, 6, 2, 0, variant=tdma.TDMA_VARIANT_FUSED, axis=tdma.TDMA_AXIS_X, periodic=1) as plan:
        plan.solve_host(*host, xh)
    check(a, b, c, d, xh, "x", True)


@pytest.mark.parametrize("opts,periodic", [(dict(variant=tdma.TDMA_VARIANT_FUSED), 1), (dict(variant=tdma.TDMA_VARIANT_PIPELINED), 0),
                                           (dict(variant=tdma.TDMA_VARIANT_PIPELINED), 1), (dict(variant=tdma.TDMA_VARIANT_STAGED), 0),
                                           (dict(), 0)], ids=["fused_cyclic", "pipelined", "pipelined_cyclic", "staged", "auto"])
@pytest.mark.parametrize("chunk", [0, 5])
def test_solve_host_on_z_sweeps(opts, periodic, chunk):
    """tdma_solve_host of a z sweep: chunks of y-slices (strided copies), each solved by a plan of its own;
    host_chunk = 5 gives 4 chunks with a ragged last one (17 = 3 * 5 + 2).  Against the oracle and, to
    rounding, against the device solve."""
    nz, ny, nx = 64, 17, 48
    a, b, c, d = tdma_inputs.dominant_random(nx, ny, nz, 63, "cpu")
    host = [t.pin_memory() for t in (a, b, c, d)]
    xh = torch.full_like(d, float("nan")).pin_memory()
    with tdma.Plan(nx, ny, nz, 4, 2, axis=tdma.TDMA_AXIS_Z, periodic=periodic, host_chunk=chunk, **opts) as plan:
        plan.solve_host(*host, xh)
        plan.solve_host(*host, xh)                       # second call: staging and chunk plans are reused
        xd = torch.full_like(d, float("nan"), device=dev())
        plan.solve(*[t.to(dev()) for t in (a, b, c, d)], xd)
        torch.cuda.synchronize()
    check(a, b, c, d, xh, "z", bool(periodic))
    assert float((xh - xd.cpu()).abs().max() / xh.abs().max()) <= 1e-13
