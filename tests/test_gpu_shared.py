"""shared-coefficient / complex-RHS lines -- the CUDA
path (tdma_solve_shared through the C ABI) against oracle.solve_y_shared, element by element on
the same seeded inputs.  Tolerance as for the general path (G9): per line and per component
E = ||x - x_or||_inf / ||x_or||_inf <= 1e-11, against the long-double oracle on the weakly
dominant Poisson coefficients of cfg 2 / cfg 3."""
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


def as_lines(x):
    """(nz, ny, nx) real or complex -> real (nz, ny, nx * ncomp): every component is a line."""
    x = np.ascontiguousarray(x)
    if np.iscomplexobj(x):
        return x.view(np.float64).reshape(x.shape[0], x.shape[1], -1)
    return x


def gpu_solve_shared(w, P=1, x=None, **opts):
    dv = dev()
    t = [v.to(dv) for v in (w.a_y, w.b0_y, w.c_y, w.sx, w.sz, w.d)]
    out = torch.full_like(t[5], float("nan")) if x is None else x
    with tdma.Plan(w.nx, w.ny, w.nz, P, 0, **opts) as plan:
        plan.solve_shared(*t[:5], t[5], out, pin00=w.pin00)
        torch.cuda.synchronize()
        info = {k: plan.get(getattr(tdma, "TDMA_GET_SHARED_" + k.upper()))
                for k in ("lines", "cluster", "leaf_rows", "threads", "slots", "fill")}
    return out, info


def oracle_shared(w, precision):
    arrs = [v.cpu().numpy() for v in (w.a_y, w.b0_y, w.c_y, w.sx, w.sz, w.d)]
    return oracle.solve_y_shared(*arrs, pin00=w.pin00, precision=precision)


def check(w, x, precision="ld"):
    xn = x.cpu().numpy()
    assert np.isfinite(as_lines(xn)).all()
    ref = oracle_shared(w, precision)
    E = oracle.normwise_error(as_lines(xn), as_lines(ref)).max()
    assert E <= TOL_E, "normwise error %.3e" % E
    return E


def random_shared(nz, ny, nx, cplx, seed):
    """Strictly dominant shared-coefficient case (the recipe of the oracle pins): a, c ~ U(-1,1),
    b0 ~ 2.5 + U(0,1), shifts <= 0 so that b >= 2.5."""
    g = torch.Generator().manual_seed(seed)
    u = lambda n, lo, hi: lo + (hi - lo) * torch.rand(n, dtype=torch.float64, generator=g)
    d = torch.randn((nz, ny, nx), dtype=torch.float64, generator=g)
    if cplx:
        d = torch.complex(d, torch.randn((nz, ny, nx), dtype=torch.float64, generator=g))
    return tdma_inputs.SharedWorkload("random_shared", nx, ny, nz, u(ny, -1, 1), u(ny, 2.5, 3.5), u(ny, -1, 1),
                                      -u(nx, 0, 2), -u(nz, 0, 2), d, pin00=False)


@pytest.mark.parametrize("cplx", [False, True], ids=["f64", "c128"])
@pytest.mark.parametrize("name,nz", [("cfg2_poisson", 6), ("cfg3_weak", 16)])
def test_poisson_shared_slab(name, nz, cplx):
    """z-slab of cfg 2 / cfg 3 at full nx, ny in the automatic tiling (cfg 3: main + fill launch)."""
    w = tdma_inputs.make_shared_workload(name, cplx, nz=nz)
    x, info = gpu_solve_shared(w)
    check(w, x, "ld")
    assert x.cpu().numpy()[0, 0, 0] == 0.0                     # pinned mean mode: x_0 = d_0 = 0
    if name == "cfg3_weak":
        assert info["cluster"] >= 2 and info["leaf_rows"] == (32 if not cplx else 16)


@pytest.mark.parametrize("cplx", [False, True], ids=["f64", "c128"])
@pytest.mark.parametrize("ny,opts", [
    (16, {}), (32, {}), (64, {}), (128, dict(shared_leaf_rows=4)), (128, dict(shared_leaf_rows=8)),
    (256, dict(shared_cluster=1)), (256, dict(shared_cluster=2)), (256, dict(shared_cluster=4, shared_leaf_rows=8)),
    (512, dict(shared_cluster=2)), (512, dict(shared_cluster=8, shared_leaf_rows=16)),
    (1024, dict(shared_cluster=2)), (1024, dict(shared_cluster=4, shared_slots=2)),
    (1024, dict(shared_cluster=8, shared_leaf_rows=8)),
    (256, dict(shared_leaf_rows=32)), (512, dict(shared_cluster=1, shared_leaf_rows=32)),
    (1024, dict(shared_cluster=2, shared_leaf_rows=32)), (1024, dict(shared_cluster=4, shared_leaf_rows=32)),
    # 3 * 2^k and 5 * 2^k line lengths: leaves of 12 / 24 and 10 / 20 rows
    (24, {}), (48, {}), (96, {}), (192, {}), (384, {}), (768, {}), (1536, {}), (3072, {}), (40, {}), (160, {}), (320, {}),
    (640, {}), (1280, {}), (768, dict(shared_leaf_rows=12)), (640, dict(shared_leaf_rows=10)),
    (768, dict(shared_cluster=8)), (1280, dict(shared_cluster=4)),
])
def test_tilings_and_ragged_x(ny, opts, cplx):
    """Every tiling the kernel is instantiated for, nx not a multiple of the tile width (the last
    x tile is clipped by TMA), several tiles per cluster."""
    w = random_shared(5, ny, 88, cplx, seed=ny + (7 if cplx else 0))
    x, info = gpu_solve_shared(w, **opts)
    check(w, x, "f64")
    assert info["threads"] > 0                               # the tiled kernel, not the one-thread-per-line kernel
    for key, name in (("shared_cluster", "cluster"), ("shared_leaf_rows", "leaf_rows"), ("shared_slots", "slots")):
        if key in opts:
            assert info[name] == opts[key]
    if ny % 3 == 0:
        assert info["leaf_rows"] in (12, 24)
    if ny % 5 == 0:
        assert info["leaf_rows"] in (10, 20)


@pytest.mark.parametrize("cplx", [False, True], ids=["f64", "c128"])
@pytest.mark.parametrize("lines", [0, 1])
def test_wide_tiles(lines, cplx):
    """256-byte row segments (32 real / 16 complex cells per tile row)."""
    w = random_shared(3, 512, 96, cplx, seed=11)
    x, info = gpu_solve_shared(w, shared_lines=(32 if not cplx else 16) if lines else 0)
    check(w, x, "f64")
    assert info["lines"] == ((32 if not cplx else 16) if lines else (16 if not cplx else 8))


@pytest.mark.parametrize("cplx", [False, True], ids=["f64", "c128"])
def test_in_place_and_repeatable(cplx):
    """x may alias d; repeated solves give the same bits (races show up as differing bits)."""
    w = random_shared(24, 1024, 64, cplx, seed=3)
    x1, _ = gpu_solve_shared(w)
    x2, _ = gpu_solve_shared(w)
    assert torch.equal(torch.view_as_real(x1) if cplx else x1, torch.view_as_real(x2) if cplx else x2)
    dcopy = w.d.clone().to(dev())
    t = [v.to(dev()) for v in (w.a_y, w.b0_y, w.c_y, w.sx, w.sz)]
    with tdma.Plan(w.nx, w.ny, w.nz, 1, 0) as plan:
        plan.solve_shared(*t, dcopy, dcopy)
        torch.cuda.synchronize()
    assert torch.equal(torch.view_as_real(dcopy) if cplx else dcopy, torch.view_as_real(x1) if cplx else x1)
    check(w, x1, "f64")


def test_complex_components_are_independent_real_solves():
    """re / im of the complex solve equal, bit for bit, what the REAL shared solve gives for each
    component in the same tiling family?  No: tilings differ, so compare within tolerance, and
    check that a purely real d gives an exactly zero imaginary part."""
    w = random_shared(4, 256, 32, True, seed=5)
    xc, _ = gpu_solve_shared(w)
    for part in ("real", "imag"):
        wr = tdma_inputs.SharedWorkload("part", w.nx, w.ny, w.nz, w.a_y, w.b0_y, w.c_y, w.sx, w.sz,
                                        getattr(w.d, part).contiguous(), False)
        xr, _ = gpu_solve_shared(wr)
        ref = getattr(xc, part).cpu().numpy()
        assert oracle.normwise_error(xr.cpu().numpy(), ref).max() <= TOL_E
    wz = tdma_inputs.SharedWorkload("realonly", w.nx, w.ny, w.nz, w.a_y, w.b0_y, w.c_y, w.sx, w.sz,
                                    torch.complex(w.d.real, torch.zeros_like(w.d.real)), False)
    xz, _ = gpu_solve_shared(wz)
    assert float(xz.imag.abs().max()) == 0.0


def test_matches_general_path_on_materialised_arrays():
    """Same systems through tdma_solve with a, b, c materialised (b formed as b0 - (sx + sz))."""
    w = random_shared(4, 512, 64, False, seed=9)
    dv = dev()
    nz, ny, nx = w.nz, w.ny, w.nx
    a = w.a_y.view(1, ny, 1).expand(nz, ny, nx).contiguous().to(dv)
    c = w.c_y.view(1, ny, 1).expand(nz, ny, nx).contiguous().to(dv)
    b = (w.b0_y.view(1, ny, 1) - (w.sx.view(1, 1, nx) + w.sz.view(nz, 1, 1))).contiguous().to(dv)
    d = w.d.to(dv)
    xg = torch.empty_like(d)
    with tdma.Plan(nx, ny, nz, 8, 0) as plan:
        plan.solve(a, b, c, d, xg)
        torch.cuda.synchronize()
    xs, _ = gpu_solve_shared(w)
    assert oracle.normwise_error(xs.cpu().numpy(), xg.cpu().numpy()).max() <= TOL_E


def test_requested_tilings_that_do_not_fit_fail_loudly():
    """A tiling asked for through the shared_* options is never replaced by another kernel: shapes it does
    not fit are refused (without such a request the one-thread-per-line kernel takes them, see
    test_line_kernel_takes_every_shape)."""
    dv = dev()
    def attempt(nx, ny, cplx, **opts):
        w = random_shared(2, ny, nx, cplx, seed=1)
        return gpu_solve_shared(w, **opts)
    with pytest.raises(tdma.TdmaError) as e1:
        attempt(32, 24, False, shared_leaf_rows=8)   # 24 rows: no power-of-two tree of 8-row leaves
    assert e1.value.status == tdma.TDMA_ERR_UNSUPPORTED
    with pytest.raises(tdma.TdmaError) as e2:
        attempt(33, 64, False, shared_cluster=1)     # odd nx, real: 8-byte global strides
    assert e2.value.status == tdma.TDMA_ERR_UNSUPPORTED
    attempt(33, 64, True, shared_cluster=1)          # complex cells are 16 bytes: fine
    w = random_shared(2, 64, 32, False, seed=1)
    t = [v.to(dv) for v in (w.a_y, w.b0_y, w.c_y, w.sx, w.sz, w.d)]
    with tdma.Plan(32, 64, 2, 1, 0, variant=tdma.TDMA_VARIANT_FUSED, periodic=1) as plan:
        with pytest.raises(tdma.TdmaError):               # the pinned mean mode belongs to plain lines
            plan.solve_shared(*t, torch.empty_like(t[5]), pin00=True)
    with tdma.Plan(64, 32, 2, 1, 0, variant=tdma.TDMA_VARIANT_FUSED, axis=tdma.TDMA_AXIS_X, shared_leaf_rows=16) as plan:
        with pytest.raises(tdma.TdmaError) as e3:         # the tiled x sweep takes real right-hand sides only
            tdma.tdma_solve_shared(plan.handle, *t[:5], 2, 0, t[5], torch.empty_like(t[5]))
        assert e3.value.status == tdma.TDMA_ERR_UNSUPPORTED
    # x lines of 40 cells are not whole 16-cell leaves
    g = torch.Generator().manual_seed(3)
    rnd = lambda *shape: torch.rand(*shape, dtype=torch.float64, generator=g).to(dv)
    with tdma.Plan(40, 32, 2, 1, 0, axis=tdma.TDMA_AXIS_X, shared_leaf_rows=16) as plan:
        assert plan.get(tdma.TDMA_GET_VARIANT) == tdma.TDMA_VARIANT_PIPELINED
        with pytest.raises(tdma.TdmaError) as e4:
            plan.solve_shared(rnd(40) - 0.5, rnd(40) + 3.0, rnd(40) - 0.5, -rnd(32), -rnd(2), rnd(2, 32, 40),
                              torch.empty(2, 32, 40, dtype=torch.float64, device=dv))
        assert e4.value.status == tdma.TDMA_ERR_UNSUPPORTED


def shared_case(axis, shape, cplx, seed):
    """1-D coefficients, shifts and d of a strictly dominant shared-coefficient case along `axis`, and the
    materialised (a, b, c) with the diagonal formed as the kernels form it, b0 - (s_lane + s_slice)."""
    nz, ny, nx = shape
    n, lanes, nsl = {"y": (ny, nx, nz), "z": (nz, nx, ny), "x": (nx, ny, nz)}[axis]
    g = torch.Generator().manual_seed(seed)
    u = lambda k, lo, hi: lo + (hi - lo) * torch.rand(k, dtype=torch.float64, generator=g)
    a1, c1, b01 = u(n, -1, 1), u(n, -1, 1), u(n, 2.5, 3.5)
    s_lane, s_slice = -u(lanes, 0, 2), -u(nsl, 0, 2)
    d = torch.randn(shape, dtype=torch.float64, generator=g)
    if cplx:
        d = torch.complex(d, torch.randn(shape, dtype=torch.float64, generator=g))
    line = {"y": (1, n, 1), "z": (n, 1, 1), "x": (1, 1, n)}[axis]
    lane = {"y": (1, 1, lanes), "z": (1, 1, lanes), "x": (1, lanes, 1)}[axis]
    slc = {"y": (nsl, 1, 1), "z": (1, nsl, 1), "x": (nsl, 1, 1)}[axis]
    def materialise(uniform):
        shift = torch.zeros(shape, dtype=torch.float64) if uniform else (s_lane.view(lane) + s_slice.view(slc)).expand(shape)
        a = a1.view(line).expand(shape).contiguous().numpy()
        c = c1.view(line).expand(shape).contiguous().numpy()
        b = (b01.view(line) - shift).contiguous().numpy()
        return a, b, c
    return (a1, b01, c1, s_lane, s_slice, d), materialise


def check_axis(a, b, c, d, x, axis, periodic):
    xn = x.cpu().numpy()
    ax = {"y": 1, "z": 0, "x": 2}[axis]
    for part in (("real", "imag") if np.iscomplexobj(xn) else (None,)):
        dn = np.ascontiguousarray(getattr(d.numpy(), part)) if part else d.numpy()
        xp = getattr(xn, part) if part else xn
        if periodic and a.shape[ax] == 2:
            # two-row ring, by Cramer's rule: [[b_0, a_0 + c_0], [a_1 + c_1, b_1]] x = d  (the oracle's
            # Sherman-Morrison form needs n >= 3)
            t = lambda v, r: np.take(v, r, axis=ax)
            m01, m10 = t(a, 0) + t(c, 0), t(a, 1) + t(c, 1)
            det = t(b, 0) * t(b, 1) - m01 * m10
            ref = np.stack([(t(dn, 0) * t(b, 1) - m01 * t(dn, 1)) / det, (t(b, 0) * t(dn, 1) - m10 * t(dn, 0)) / det], axis=ax)
        else:
            ref = oracle.solve_axis(a, b, c, dn, axis, periodic)
        err = (np.max(np.abs(xp - ref), axis=ax) / np.max(np.abs(ref), axis=ax)).max()
        assert np.isfinite(xp).all() and err <= TOL_E, err


@pytest.mark.parametrize("cplx", [False, True], ids=["f64", "c128"])
@pytest.mark.parametrize("periodic", [False, True], ids=["plain", "cyclic"])
@pytest.mark.parametrize("axis,shape", [
    ("y", (3, 28, 32)), ("y", (4, 100, 33)), ("y", (2, 200, 7)), ("y", (5, 2, 9)), ("y", (3, 3, 1)), ("y", (2, 1000, 64)),
    ("z", (100, 3, 33)), ("z", (37, 5, 16)), ("x", (3, 9, 40)), ("x", (2, 5, 115)), ("x", (2, 3, 64))])
def test_line_kernel_takes_every_shape(axis, shape, periodic, cplx):
    """tdma_solve_shared on what the tiled TMA kernel refuses -- line lengths without a power-of-two tree of
    4- .. 32-row leaves, odd nx with real cells, complex cells along x: the one-thread-per-line kernel,
    y / z / x sweeps, plain and cyclic lines, per-line shifts and the uniform matrix, in place."""
    if axis == "x" and shape[2] % 16 == 0 and not cplx:
        pytest.skip("the tiled x-sweep kernel takes this one")
    (a1, b01, c1, s_lane, s_slice, d), materialise = shared_case(axis, shape, cplx, seed=sum(shape))
    nz, ny, nx = shape
    dv = dev()
    opts = dict(periodic=1 if periodic else 0)
    if axis != "y":
        opts["axis"] = {"z": tdma.TDMA_AXIS_Z, "x": tdma.TDMA_AXIS_X}[axis]
    coef = [t.to(dv) for t in (a1, b01, c1)]
    x = torch.full_like(d, float("nan")).to(dv)
    xu = d.clone().to(dv)                                     # the uniform-matrix solve runs in place
    with tdma.Plan(nx, ny, nz, 1, 0, **opts) as plan:
        plan.solve_shared(*coef, s_lane.to(dv), s_slice.to(dv), d.to(dv), x)
        assert plan.get(tdma.TDMA_GET_SHARED_LINE_KERNEL) == 1 and plan.get(tdma.TDMA_GET_SHARED_THREADS) == 0
        plan.solve_shared(*coef, None, None, xu, xu)
        torch.cuda.synchronize()
    check_axis(*materialise(False), d, x, axis, periodic)
    check_axis(*materialise(True), d, xu, axis, periodic)


def test_line_kernel_pinned_row_and_unaligned_arrays():
    """pin00 on the line kernel (ny = 100), and d / x that are only 8-byte aligned on a shape the tiled kernel
    would take (ny = 64): the same systems through both kernels agree to rounding."""
    w = random_shared(3, 100, 18, False, seed=8)
    w.pin00 = True
    x, _ = gpu_solve_shared(w)
    check(w, x, "f64")
    w = random_shared(4, 64, 32, True, seed=9)
    dv = dev()
    t = [v.to(dv) for v in (w.a_y, w.b0_y, w.c_y, w.sx, w.sz)]
    x_tiled, _ = gpu_solve_shared(w)
    n = w.nz * w.ny * w.nx
    buf_d = torch.empty(2 * n + 1, dtype=torch.float64, device=dv)
    buf_x = torch.full((2 * n + 1,), float("nan"), dtype=torch.float64, device=dv)
    buf_d[1:].copy_(torch.view_as_real(w.d.to(dv)).reshape(-1))
    with tdma.Plan(w.nx, w.ny, w.nz, 1, 0) as plan:
        tdma.tdma_solve_shared(plan.handle, *t, 2, 0, buf_d[1:], buf_x[1:])
        torch.cuda.synchronize()
        assert plan.get(tdma.TDMA_GET_SHARED_LINE_KERNEL) == 1
    xl = torch.view_as_complex(buf_x[1:].reshape(w.nz, w.ny, w.nx, 2).clone())
    check(w, xl, "f64")
    assert oracle.normwise_error(as_lines(xl.cpu().numpy()), as_lines(x_tiled.cpu().numpy())).max() <= 1e-13


@pytest.mark.parametrize("cplx", [False, True], ids=["f64", "c128"])
def test_fill_launch_is_repeatable(cplx):
    """cfg-3 slab in the automatic tiling (main launch + fill launch with 512-thread CTAs), solved
    repeatedly: every solve must match the reference.  (Regression: stage B once wrote its result
    over node rows that slower warps of the same CTA were still sending to the peer CTAs.)"""
    w = tdma_inputs.make_shared_workload("cfg3_weak", cplx, nz=16)
    ref = as_lines(oracle_shared(w, "ld"))
    for rep in range(8):
        x, info = gpu_solve_shared(w, shared_cluster=4, shared_leaf_rows=16)     # clusters of 4 leave SMs to the fill launch
        assert info["fill"] > 0
        E = oracle.normwise_error(as_lines(x.cpu().numpy()), ref).max()
        assert E <= TOL_E, "solve %d: normwise error %.3e (fill %d)" % (rep, E, info["fill"])


@pytest.mark.parametrize("cplx", [False, True], ids=["f64", "c128"])
def test_cfg3_shared_full_size_sampled(cplx):
    """The launch configuration bench.py times for the shared-coefficient workloads: cfg 3 at FULL
    size (1024^3 cells, complex: 2 x 16 GiB), one persistent launch (plus the fill launch where the
    tiling has one), sampled z-slices against the long-double reference slice by slice."""
    free, _ = torch.cuda.mem_get_info()
    need = 1024 ** 3 * 8 * (2 if cplx else 1) * 2 * 1.15
    if free < need:
        pytest.skip("needs %.0f GB of device memory" % (need / 1e9))
    dv = dev()
    w = tdma_inputs.make_shared_workload("cfg3_weak", cplx, device=dv)
    x = torch.full_like(w.d, float("nan"))
    with tdma.Plan(w.nx, w.ny, w.nz, 1, 0) as plan:
        plan.solve_shared(w.a_y, w.b0_y, w.c_y, w.sx, w.sz, w.d, x, pin00=True)
        torch.cuda.synchronize()
        fill = plan.get(tdma.TDMA_GET_SHARED_FILL)
    picks = {0, 1, 511, 777, w.nz - 1}
    if fill > 0:
        picks |= {w.nz - fill - 1, w.nz - fill, w.nz - fill // 2 - 1}
    host = [t.cpu().numpy() for t in (w.a_y, w.b0_y, w.c_y, w.sx)]
    for k in sorted(picks):
        ref = oracle.solve_y_shared(*host, w.sz[k:k + 1].cpu().numpy(), w.d[k:k + 1].cpu().numpy(),
                                    pin00=(k == 0), precision="ld")
        xk = x[k:k + 1].cpu().numpy()
        assert np.isfinite(as_lines(xk)).all()
        E = oracle.normwise_error(as_lines(xk), as_lines(ref)).max()
        assert E <= TOL_E, "slice %d: normwise error %.3e" % (k, E)
    del w, x
    torch.cuda.empty_cache()


@pytest.mark.parametrize("cplx", [False, True], ids=["f64", "c128"])
@pytest.mark.parametrize("axis,periodic,shape", [
    ("y", True, (5, 256, 48)), ("y", True, (3, 1024, 40)), ("z", False, (256, 6, 48)),
    ("z", True, (512, 5, 40)), ("z", True, (64, 7, 32)), ("z", False, (1024, 3, 64)),
])
def test_shared_z_sweeps_and_cyclic_lines(axis, periodic, shape, cplx):
    """Shared coefficients along z and / or with the cyclic coupling (the matrix-sharing momentum sweeps
    of the ADI scheme): against oracle.solve_axis on the materialised arrays, whose
    diagonal is formed exactly as the kernel forms it, b0 - (sx + s_slice)."""
    nz, ny, nx = shape
    n, nsl = (nz, ny) if axis == "z" else (ny, nz)            # line length, slices
    g = torch.Generator().manual_seed(1000 + n + nsl)
    u = lambda k, lo, hi: lo + (hi - lo) * torch.rand(k, dtype=torch.float64, generator=g)
    a1, c1, b01 = u(n, -1, 1), u(n, -1, 1), u(n, 2.5, 3.5)
    sx, ss = -u(nx, 0, 2), -u(nsl, 0, 2)
    d = torch.randn((nz, ny, nx), dtype=torch.float64, generator=g)
    if cplx:
        d = torch.complex(d, torch.randn((nz, ny, nx), dtype=torch.float64, generator=g))
    dv = dev()
    x = torch.full_like(d, float("nan")).to(dv)
    opts = dict(axis=tdma.TDMA_AXIS_Z if axis == "z" else tdma.TDMA_AXIS_Y, periodic=1 if periodic else 0)
    with tdma.Plan(nx, ny, nz, 1, 0, **opts) as plan:
        plan.solve_shared(*[t.to(dv) for t in (a1, b01, c1, sx, ss)], d.to(dv), x)
        torch.cuda.synchronize()
    # materialise: the line axis is z (dim 0) or y (dim 1) of the (nz, ny, nx) arrays
    line = (n, 1, 1) if axis == "z" else (1, n, 1)
    sl = (1, nsl, 1) if axis == "z" else (nsl, 1, 1)
    a = a1.view(line).expand(nz, ny, nx).contiguous().numpy()
    c = c1.view(line).expand(nz, ny, nx).contiguous().numpy()
    b = (b01.view(line) - (sx.view(1, 1, nx) + ss.view(sl))).expand(nz, ny, nx).contiguous().numpy()
    xn = x.cpu().numpy()
    ax = 0 if axis == "z" else 1
    for part in (("real", "imag") if cplx else (None,)):
        dn = getattr(d, part).contiguous().numpy() if part else d.numpy()
        xp = getattr(xn, part) if part else xn
        ref = oracle.solve_axis(a, b, c, dn, axis, periodic)
        err = (np.max(np.abs(xp - ref), axis=ax) / np.max(np.abs(ref), axis=ax)).max()
        assert np.isfinite(xp).all() and err <= TOL_E, err


@pytest.mark.parametrize("periodic", [False, True], ids=["plain", "cyclic"])
@pytest.mark.parametrize("leaf", [0, 16], ids=["auto", "leaf16"])
@pytest.mark.parametrize("shape", [(3, 40, 256), (2, 37, 512), (5, 16, 64), (2, 130, 1024), (4, 9, 16), (2, 24, 2048)])
def test_shared_x_sweeps(shape, periodic, leaf):
    """Shared coefficients along x (lines along the contiguous axis: the third momentum sweep of the ADI
    scheme), real right-hand sides: a_y, b0_y, c_y hold nx entries, sx one shift per
    line of a slice (ny), sz one per slice.  Ragged line tiles (ny not a multiple of 16), one to
    several CTAs per line, the fill tiling at 1024 cells.  Against oracle.solve_axis on the
    materialised arrays."""
    nz, ny, nx = shape
    g = torch.Generator().manual_seed(2000 + nx + ny)
    u = lambda k, lo, hi: lo + (hi - lo) * torch.rand(k, dtype=torch.float64, generator=g)
    a1, c1, b01 = u(nx, -1, 1), u(nx, -1, 1), u(nx, 2.5, 3.5)
    sy, sz = -u(ny, 0, 2), -u(nz, 0, 2)
    d = torch.randn((nz, ny, nx), dtype=torch.float64, generator=g)
    dv = dev()
    x = torch.full_like(d, float("nan")).to(dv)
    with tdma.Plan(nx, ny, nz, 1, 0, axis=tdma.TDMA_AXIS_X, periodic=1 if periodic else 0, shared_leaf_rows=leaf) as plan:
        for _ in range(2):
            plan.solve_shared(*[t.to(dv) for t in (a1, b01, c1, sy, sz)], d.to(dv), x)
        torch.cuda.synchronize()
        assert plan.get(tdma.TDMA_GET_SHARED_LEAF_ROWS) == (leaf if leaf else (32 if nx >= 32 else 16))
    a = a1.view(1, 1, nx).expand(nz, ny, nx).contiguous().numpy()
    c = c1.view(1, 1, nx).expand(nz, ny, nx).contiguous().numpy()
    b = (b01.view(1, 1, nx) - (sy.view(1, ny, 1) + sz.view(nz, 1, 1))).expand(nz, ny, nx).contiguous().numpy()
    xn = x.cpu().numpy()
    ref = oracle.solve_axis(a, b, c, d.numpy(), "x", periodic)
    err = (np.max(np.abs(xn - ref), axis=2) / np.max(np.abs(ref), axis=2)).max()
    assert np.isfinite(xn).all() and err <= TOL_E, err


def test_shared_x_sweep_in_place_and_pinned():
    """x = d in place, and the pinned row 0 of line (0, 0) in an x sweep."""
    nz, ny, nx = 3, 20, 128
    g = torch.Generator().manual_seed(77)
    u = lambda k, lo, hi: lo + (hi - lo) * torch.rand(k, dtype=torch.float64, generator=g)
    a1, c1, b01 = u(nx, -1, 1), u(nx, -1, 1), u(nx, 2.5, 3.5)
    sy, sz = -u(ny, 0, 2), -u(nz, 0, 2)
    d = torch.randn((nz, ny, nx), dtype=torch.float64, generator=g)
    dv = dev()
    x = d.clone().to(dv)
    with tdma.Plan(nx, ny, nz, 1, 0, axis=tdma.TDMA_AXIS_X) as plan:
        plan.solve_shared(*[t.to(dv) for t in (a1, b01, c1, sy, sz)], x, x, pin00=True)
        torch.cuda.synchronize()
    a = a1.view(1, 1, nx).expand(nz, ny, nx).contiguous().numpy()
    c = c1.view(1, 1, nx).expand(nz, ny, nx).contiguous().numpy()
    b = (b01.view(1, 1, nx) - (sy.view(1, ny, 1) + sz.view(nz, 1, 1))).expand(nz, ny, nx).contiguous().numpy()
    b[0, 0, 0] = 1.0
    c[0, 0, 0] = 0.0
    ref = oracle.solve_axis(a, b, c, d.numpy(), "x", False)
    xn = x.cpu().numpy()
    err = (np.max(np.abs(xn - ref), axis=2) / np.max(np.abs(ref), axis=2)).max()
    assert np.isfinite(xn).all() and err <= TOL_E, err


def test_cfg4_adi_full_size_in_shared_form_sampled():
    """BASELINE cfg 4 at FULL size (512^3) in the matrix-sharing form `bench.py --adi` times
    (PAPER.md:318): x periodic -> y Dirichlet -> z periodic with a = c = -alpha, b = 1 + 2 alpha as 1-D
    arrays and zero shifts; every sweep against oracle.solve_axis on sampled z-slices / y-planes."""
    w = tdma_inputs.make_workload("cfg4_adi_y", device=dev())
    dv = dev()
    alpha = float(w.meta["alpha"])
    coef = lambda n: (torch.full((n,), -alpha, dtype=torch.float64, device=dv),
                      torch.full((n,), 1.0 + 2.0 * alpha, dtype=torch.float64, device=dv),
                      torch.full((n,), -alpha, dtype=torch.float64, device=dv))
    zero = lambda n: torch.zeros(n, dtype=torch.float64, device=dv)
    src = w.d
    for axis, name, periodic, n, lanes, nsl in ((tdma.TDMA_AXIS_X, "x", 1, w.nx, w.ny, w.nz),
                                                (tdma.TDMA_AXIS_Y, "y", 0, w.ny, w.nx, w.nz),
                                                (tdma.TDMA_AXIS_Z, "z", 1, w.nz, w.nx, w.ny)):
        dst = torch.full_like(w.d, float("nan"))
        with tdma.Plan(w.nx, w.ny, w.nz, 1, 0, axis=axis, periodic=periodic) as plan:
            plan.solve_shared(*coef(n), zero(lanes), zero(nsl), src, dst)
            torch.cuda.synchronize()
            fill = plan.get(tdma.TDMA_GET_SHARED_FILL)
        assert bool(torch.isfinite(dst).all())
        picks = {0, 1, nsl // 2 + 1, nsl - 1}
        if fill > 0:
            picks |= {nsl - fill, nsl - fill - 1}
        ax = {"y": 1, "z": 0, "x": 2}[name]
        for q in sorted(picks):
            sl = (slice(None), slice(q, q + 1)) if name == "z" else (slice(q, q + 1),)
            an, bn, cn, dn, xn = [t[sl].cpu().numpy() for t in (w.a, w.b, w.c, src, dst)]
            ref = oracle.solve_axis(an, bn, cn, dn, name, bool(periodic))
            err = (np.max(np.abs(xn - ref), axis=ax) / np.max(np.abs(ref), axis=ax)).max()
            assert err <= TOL_E, (name, q, err)
        src = dst


@pytest.mark.parametrize("periodic", [False, True], ids=["plain", "cyclic"])
@pytest.mark.parametrize("axis,shape,leaf", [
    ("y", (5, 512, 48), 0), ("y", (3, 1024, 40), 0), ("y", (6, 256, 64), 16), ("y", (4, 64, 32), 0),
    ("z", (512, 5, 48), 0), ("z", (1024, 3, 64), 16), ("x", (3, 40, 512), 0), ("x", (2, 37, 1024), 0),
    ("x", (4, 20, 256), 16), ("y", (2, 2048, 32), 0),
])
def test_uniform_matrix_equals_zero_shifts(axis, shape, leaf, periodic):
    """sx = sz = NULL (the same matrix for every line: the ADI momentum sweeps): the
    matrix work is hoisted out of the tile loop; x must agree with what zero shift arrays give to
    rounding (same formulas, contracted differently), and with oracle.solve_axis within the tolerance.  One to several CTAs per line, both
    leaf sizes, ragged line tiles, the fill launch at 1024 rows."""
    nz, ny, nx = shape
    n, lanes, nsl = {"y": (ny, nx, nz), "z": (nz, nx, ny), "x": (nx, ny, nz)}[axis]
    g = torch.Generator().manual_seed(3000 + n + nsl)
    u = lambda k, lo, hi: lo + (hi - lo) * torch.rand(k, dtype=torch.float64, generator=g)
    a1, c1, b01 = u(n, -1, 1), u(n, -1, 1), u(n, 2.5, 3.5)
    d = torch.randn((nz, ny, nx), dtype=torch.float64, generator=g)
    dv = dev()
    ax = {"y": tdma.TDMA_AXIS_Y, "z": tdma.TDMA_AXIS_Z, "x": tdma.TDMA_AXIS_X}[axis]
    coef = [t.to(dv) for t in (a1, b01, c1)]
    zl, zs = torch.zeros(lanes, dtype=torch.float64, device=dv), torch.zeros(nsl, dtype=torch.float64, device=dv)
    xu, xz = [torch.full_like(d, float("nan")).to(dv) for _ in range(2)]
    with tdma.Plan(nx, ny, nz, 1, 0, axis=ax, periodic=1 if periodic else 0, shared_lines=16,
                   shared_leaf_rows=leaf) as plan:
        for _ in range(2):
            plan.solve_shared(*coef, None, None, d.to(dv), xu)
        torch.cuda.synchronize()
        cfg_u = [plan.get(q) for q in (tdma.TDMA_GET_SHARED_LINES, tdma.TDMA_GET_SHARED_CLUSTER, tdma.TDMA_GET_SHARED_LEAF_ROWS)]
        plan.solve_shared(*coef, zl, zs, d.to(dv), xz)
        torch.cuda.synchronize()
        cfg_z = [plan.get(q) for q in (tdma.TDMA_GET_SHARED_LINES, tdma.TDMA_GET_SHARED_CLUSTER, tdma.TDMA_GET_SHARED_LEAF_ROWS)]
    line = {"y": (1, n, 1), "z": (n, 1, 1), "x": (1, 1, n)}[axis]
    a = a1.view(line).expand(nz, ny, nx).contiguous().numpy()
    b = b01.view(line).expand(nz, ny, nx).contiguous().numpy()
    c = c1.view(line).expand(nz, ny, nx).contiguous().numpy()
    ref = oracle.solve_axis(a, b, c, d.numpy(), axis, periodic)
    xn = xu.cpu().numpy()
    dim = {"y": 1, "z": 0, "x": 2}[axis]
    err = (np.max(np.abs(xn - ref), axis=dim) / np.max(np.abs(ref), axis=dim)).max()
    assert np.isfinite(xn).all() and err <= TOL_E, err
    assert cfg_u[0] == 16 and cfg_u[2] in (16, 32)
    tol = 1e-13 if cfg_u == cfg_z else TOL_E        # same tiling: the same formulas in the same order
    assert (np.max(np.abs(xn - xz.cpu().numpy()), axis=dim) / np.max(np.abs(ref), axis=dim)).max() <= tol


def test_uniform_matrix_fallback_and_errors():
    """Complex cells and shapes outside the uniform-matrix build run the general form with plan-owned
    zero shifts; pin00 and a single NULL shift array are refused."""
    dv = dev()
    nz, ny, nx = 3, 128, 24
    g = torch.Generator().manual_seed(5)
    u = lambda k, lo, hi: lo + (hi - lo) * torch.rand(k, dtype=torch.float64, generator=g)
    a1, c1, b01 = u(ny, -1, 1), u(ny, -1, 1), u(ny, 2.5, 3.5)
    d = torch.complex(torch.randn((nz, ny, nx), dtype=torch.float64, generator=g),
                      torch.randn((nz, ny, nx), dtype=torch.float64, generator=g))
    coef = [t.to(dv) for t in (a1, b01, c1)]
    zx, zz = torch.zeros(nx, dtype=torch.float64, device=dv), torch.zeros(nz, dtype=torch.float64, device=dv)
    x1, x2 = [torch.full_like(d, float("nan")).to(dv) for _ in range(2)]
    with tdma.Plan(nx, ny, nz, 1, 0) as plan:
        plan.solve_shared(*coef, None, None, d.to(dv), x1)          # complex: general form, zero shifts
        plan.solve_shared(*coef, zx, zz, d.to(dv), x2)
        torch.cuda.synchronize()
        assert torch.equal(x1, x2)
        with pytest.raises(tdma.TdmaError):
            tdma.tdma_solve_shared(plan.handle, *coef, zx, 0, 1, 0, x1.real.contiguous(), x2.real.contiguous())
        with pytest.raises(tdma.TdmaError):
            tdma.tdma_solve_shared(plan.handle, *coef, 0, 0, 1, 1, x1.real.contiguous(), x2.real.contiguous())
    # real cells, 8-row leaves forced: outside the uniform build (16- / 32-row leaves) -> general form
    dr = d.real.contiguous().to(dv)
    y1, y2 = [torch.full_like(dr, float("nan")) for _ in range(2)]
    with tdma.Plan(nx, ny, nz, 1, 0, shared_leaf_rows=8) as plan:
        plan.solve_shared(*coef, None, None, dr, y1)
        plan.solve_shared(*coef, zx, zz, dr, y2)
        torch.cuda.synchronize()
        assert plan.get(tdma.TDMA_GET_SHARED_LEAF_ROWS) == 8
    assert torch.equal(y1, y2)
