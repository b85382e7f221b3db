"""Seeded random sweep over shapes and options of tdma_solve / tdma_solve_shared (through the C ABI)
against the oracle: every case either solves within the 1e-11 tolerance of G9 or is refused at plan
creation / solve with TDMA_ERR_UNSUPPORTED -- never a wrong x, never a non-finite one, and under the AUTO
and PIPELINED variants nothing is refused (the stage pipeline takes what the TMA kernels cannot tile).
The shapes mix the line lengths the kernels tile (2^k, 3 * 2^k, 5 * 2^k), lengths they cannot, odd and
ragged nx, one-row partitions' neighbours (m = 2), ragged last batches, cyclic lines, all sweep axes."""
import numpy as np
import pytest
import torch

import oracle
import tdma_inputs
import paper_2509_03933_b200 as tdma

pytestmark = pytest.mark.gpu
TOL_E = 1e-11

POOL_N = [2, 3, 4, 6, 8, 10, 12, 16, 20, 24, 32, 40, 48, 64, 80, 96, 128, 160, 192, 256, 320, 384, 512, 640, 768,
          1024, 1536, 2048]
POOL_L = [1, 2, 3, 5, 8, 15, 16, 17, 24, 31, 32, 33, 48, 64, 100, 128, 250, 256, 510, 512, 1000, 1022, 1023, 1024]
VARIANTS = {"auto": {}, "pipelined": dict(variant=tdma.TDMA_VARIANT_PIPELINED),
            "staged": dict(variant=tdma.TDMA_VARIANT_STAGED), "fused": dict(variant=tdma.TDMA_VARIANT_FUSED),
            "fused_reg": dict(variant=tdma.TDMA_VARIANT_FUSED, fused_impl=1)}


def dev():
    return torch.device("cuda:0")


def divisors(n):
    return [p for p in range(1, n + 1) if n % p == 0 and (p == 1 or n // p >= 2)]


def draw_case(rng):
    axis = str(rng.choice(["y", "z", "x"], p=[0.5, 0.25, 0.25]))
    n = int(rng.choice(POOL_N)) if rng.rand() < 0.8 else int(rng.randint(2, 200))
    if axis == "x" and rng.rand() < 0.8:
        n = int(rng.choice([16, 32, 48, 64, 128, 256, 512, 1024, 2048]))
    P = int(rng.choice(divisors(n)))
    lanes = int(rng.choice(POOL_L)) if rng.rand() < 0.7 else int(rng.randint(1, 80))
    slices = int(rng.randint(1, max(1, min(40, (1 << 20) // (n * lanes))) + 1))
    periodic = int(rng.rand() < 0.3) if n >= 3 else 0
    vname = str(rng.choice(list(VARIANTS), p=[0.4, 0.15, 0.15, 0.2, 0.1]))
    batch = 0 if rng.rand() < 0.5 else int(rng.randint(1, slices + 1))
    shape = {"y": (slices, n, lanes), "z": (n, slices, lanes), "x": (slices, lanes, n)}[axis]
    return axis, shape, P, periodic, vname, batch


@pytest.mark.parametrize("seed", [101, 202, 303, 404])
def test_random_shapes_general_form(seed):
    rng = np.random.RandomState(seed)
    solved = refused = 0
    for it in range(60):
        axis, (nz, ny, nx), P, periodic, vname, batch = draw_case(rng)
        opts = dict(VARIANTS[vname])
        if axis != "y":
            opts["axis"] = {"z": tdma.TDMA_AXIS_Z, "x": tdma.TDMA_AXIS_X}[axis]
        if periodic:
            opts["periodic"] = 1
        tag = "seed %d case %d: axis %s shape %s P %d periodic %d %s batch %d" % (seed, it, axis, (nz, ny, nx), P,
                                                                                periodic, vname, batch)
        a, b, c, d = tdma_inputs.dominant_random(nx, ny, nz, 1000 * seed + it, dev())
        x = torch.full_like(d, float("nan"))
        try:
            with tdma.Plan(nx, ny, nz, P, batch, **opts) as plan:
                plan.solve(a, b, c, d, x)
                torch.cuda.synchronize()
        except tdma.TdmaError as e:
            assert e.status == tdma.TDMA_ERR_UNSUPPORTED, tag + ": " + str(e)
            assert vname not in ("auto", "pipelined"), tag + " refused: " + str(e)
            refused += 1
            continue
        an, bn, cn, dn, xn = [t.cpu().numpy() for t in (a, b, c, d, x)]
        assert np.isfinite(xn).all(), tag
        ref = oracle.solve_axis(an, bn, cn, dn, axis, bool(periodic))
        ax = {"y": 1, "z": 0, "x": 2}[axis]
        err = (np.max(np.abs(xn - ref), axis=ax) / np.max(np.abs(ref), axis=ax)).max()
        assert err <= TOL_E, tag + ": E = %.3e" % err
        solved += 1
    assert solved >= 30 and solved + refused == 60


def as_lines(x):
    x = np.ascontiguousarray(x)
    if np.iscomplexobj(x):
        return x.view(np.float64).reshape(x.shape[0], x.shape[1], -1)
    return x


@pytest.mark.parametrize("seed", [11, 22, 33])
def test_random_shapes_shared_form(seed):
    """tdma_solve_shared along y: real / complex cells, per-line shifts or a uniform matrix, plain or cyclic
    lines, in place or not; ny that the tiled kernel takes and ny that go to the one-thread-per-line kernel;
    odd, ragged and tiny nx.  Nothing is refused."""
    rng = np.random.RandomState(seed)
    pool_n = [4, 8, 16, 32, 48, 64, 96, 128, 192, 256, 384, 512, 640, 768, 1024, 2048, 4096]
    tiled = lines = 0
    for it in range(50):
        ny = int(rng.choice(pool_n)) if rng.rand() < 0.85 else int(rng.randint(2, 300))
        nx = int(rng.choice(POOL_L)) if rng.rand() < 0.7 else int(rng.randint(1, 80))
        nz = int(rng.randint(1, max(1, min(40, (1 << 19) // (ny * nx))) + 1))
        cplx, uniform = bool(rng.rand() < 0.4), bool(rng.rand() < 0.3)
        periodic, inplace = int(rng.rand() < 0.25) if ny >= 3 else 0, bool(rng.rand() < 0.3)
        tag = "seed %d case %d: shape %s cplx %d uniform %d periodic %d inplace %d" % (seed, it, (nz, ny, nx), cplx,
                                                                                     uniform, periodic, inplace)
        g = torch.Generator().manual_seed(100 * seed + it)
        u = lambda n, lo, hi: lo + (hi - lo) * torch.rand(n, dtype=torch.float64, generator=g)
        d = torch.randn((nz, ny, nx), dtype=torch.float64, generator=g)
        if cplx:
            d = torch.complex(d, torch.randn((nz, ny, nx), dtype=torch.float64, generator=g))
        a_y, b0_y, c_y = u(ny, -1, 1), u(ny, 2.5, 3.5), u(ny, -1, 1)
        sx, sz = -u(nx, 0, 2), -u(nz, 0, 2)
        if uniform:
            sx, sz = torch.zeros(nx, dtype=torch.float64), torch.zeros(nz, dtype=torch.float64)
        dd = d.to(dev())
        x = dd.clone() if inplace else torch.full_like(dd, float("nan"))
        with tdma.Plan(nx, ny, nz, 1, 0, **(dict(periodic=1) if periodic else {})) as plan:
            plan.solve_shared(a_y.to(dev()), b0_y.to(dev()), c_y.to(dev()), None if uniform else sx.to(dev()),
                              None if uniform else sz.to(dev()), x if inplace else dd, x)
            torch.cuda.synchronize()
            if plan.get(tdma.TDMA_GET_SHARED_LINE_KERNEL):
                lines += 1
            else:
                tiled += 1
        xn = x.cpu().numpy()
        assert np.isfinite(as_lines(xn)).all(), tag
        if periodic:                                        # the materialised cyclic lines, one component at a time
            bf = b0_y.numpy()[None, :, None] - (sx.numpy()[None, None, :] + sz.numpy()[:, None, None])
            af = np.broadcast_to(a_y.numpy()[None, :, None], bf.shape).copy()
            cf = np.broadcast_to(c_y.numpy()[None, :, None], bf.shape).copy()
            dn = d.numpy()
            comps = [np.ascontiguousarray(dn.real), np.ascontiguousarray(dn.imag)] if cplx else [dn]
            sols = [oracle.solve_axis(af, bf, cf, q, "y", True) for q in comps]
            ref = sols[0] + 1j * sols[1] if cplx else sols[0]
        else:
            ref = oracle.solve_y_shared(a_y.numpy(), b0_y.numpy(), c_y.numpy(), sx.numpy(), sz.numpy(), d.numpy(),
                                        pin00=False, precision="f64")
        E = oracle.normwise_error(as_lines(xn), as_lines(ref)).max()
        assert E <= TOL_E, tag + ": E = %.3e" % E
    assert tiled >= 10 and lines >= 5 and tiled + lines == 50
