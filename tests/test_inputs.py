"""The seeded generators: determinism, chunk-invariance, value distributions, and the structural
properties DESIGN.md's input recipe promises (strict dominance of cfg 1/4/5, Poisson row sums)."""
import math

import numpy as np
import pytest
import torch

import tdma_inputs as ti


def test_splitmix_matches_big_integer_reference():
    idx = torch.tensor([0, 1, 2, 12345, 2 ** 40 + 7, 2 ** 33 - 1], dtype=torch.int64)
    for seed, stream in [(0, 0), (4, 3), (123, 1000)]:
        got = ti._splitmix(idx, seed, stream)
        for n, g in zip(idx.tolist(), got.tolist()):
            ref = ti.splitmix64_reference(n, seed, stream)
            assert (g & ((1 << 64) - 1)) == ref


def test_uniform_range_and_moments():
    idx = torch.arange(1 << 18, dtype=torch.int64)
    u = ti.uniform01(idx, 0, 0)
    assert u.dtype == torch.float64
    assert float(u.min()) >= 0.0 and float(u.max()) < 1.0
    assert abs(float(u.mean()) - 0.5) < 5e-3
    assert abs(float(u.var()) - 1.0 / 12.0) < 2e-3
    z = ti.normal01(idx, 1, 0)
    assert abs(float(z.mean())) < 1e-2 and abs(float(z.std()) - 1.0) < 1e-2
    # streams are independent draws
    assert abs(float(((u - 0.5) * (ti.uniform01(idx, 0, 1) - 0.5)).mean())) < 1e-3


def test_chunked_generation_is_slice_consistent():
    full = ti.make_workload("cfg1_tiny")
    part = ti.make_workload("cfg1_tiny", nz=5, k_offset=40)
    for name in "abcd":
        assert torch.equal(getattr(full, name)[40:45], getattr(part, name))
    w3 = ti.make_workload("cfg3_weak", nx=32, nz=2, k_offset=7)
    w3b = ti.make_workload("cfg3_weak", nx=32, nz=1, k_offset=8)
    for name in "abcd":
        assert torch.equal(getattr(w3, name)[1:2], getattr(w3b, name))


def test_cfg1_recipe():
    w = ti.make_workload("cfg1_tiny")
    assert (w.nx, w.ny, w.nz, w.P, w.batch) == (64, 64, 64, 4, 0)
    assert w.a.shape == (64, 64, 64) and w.a.is_contiguous()
    assert float(w.a.abs().max()) < 1 and float(w.c.abs().max()) < 1 and float(w.d.abs().max()) < 1
    margin = w.b - w.a.abs() - w.c.abs()
    assert float(margin.min()) >= 2.0 and float(margin.max()) < 3.0
    # determinism: a fixed value of the seed-0 stream
    assert w.a[0, 0, 0].item() == 2.0 * (ti.splitmix64_reference(0, 0, 0) >> 11) * 2.0 ** -53 - 1.0


def test_poisson_coefficients_structure():
    for beta in (None, 2.0):
        a_y, c_y = ti.poisson_y_coefficients(64, beta)
        assert a_y[0] == 0 and c_y[-1] == 0
        assert (a_y[1:] > 0).all() and (c_y[:-1] > 0).all()
        # d2/dy2 annihilates constants: row sums of (a, -(a+c), c) vanish by construction,
        # and is exact on linear functions of the cell centres in the interior
        q = torch.arange(65, dtype=torch.float64)
        xi = -1 + 2 * q / 64
        yf = xi if beta is None else torch.tanh(beta * xi) / math.tanh(beta)
        yc = 0.5 * (yf[1:] + yf[:-1])
        lin = a_y[1:-1] * yc[:-2] - (a_y[1:-1] + c_y[1:-1]) * yc[1:-1] + c_y[1:-1] * yc[2:]
        assert float(lin.abs().max()) < 1e-9 * float(a_y.max())
    a_u, c_u = ti.poisson_y_coefficients(1024, None)
    h = 2.0 / 1024
    assert torch.allclose(a_u[1:], torch.full((1023,), 1 / h ** 2, dtype=torch.float64), rtol=1e-12)


def test_cfg2_recipe_small():
    w = ti.make_workload("cfg2_poisson", nx=16, nz=4)
    assert w.P == 8 and w.ny == 256
    # pinned (0,0) line
    assert w.b[0, 0, 0] == 1 and w.c[0, 0, 0] == 0 and w.d[0, 0, 0] == 0
    # all other lines: b = -(a+c) - k^2 with k^2 > 0  => strictly dominant, b < 0
    a0 = w.a.clone(); a0[:, 0, :] = 0
    c0 = w.c.clone(); c0[:, -1, :] = 0
    slack = w.b.abs() - a0.abs() - c0.abs()
    slack[0, :, 0] = 1.0
    assert float(slack.min()) > 0
    kx1 = (2 * math.sin(math.pi / 16) / (2 * math.pi / 16)) ** 2
    assert abs(float(slack[0, 5, 1]) - kx1) < 1e-9 * float(w.b[0, 5, 1].abs())


def test_cfg4_recipe_small():
    w = ti.make_workload("cfg4_adi_y", nx=8, nz=2)
    al = w.meta["alpha"]
    assert 0.1 <= al <= 10.0
    assert torch.all(w.a == -al) and torch.all(w.c == -al) and torch.all(w.b == 1 + 2 * al)
    assert float(w.d.abs().max()) < 1


def test_identity_system():
    a, b, c, d = ti.identity_system(4, 8, 2, 0)
    assert torch.all(a == 0) and torch.all(c == 0) and torch.all(b == 1)
    a, b, c, d = ti.identity_system(4, 8, 2, 0, diagonal_only=True)
    assert float(b.min()) >= 1 and float(b.max()) < 2


def test_shared_form_of_the_poisson_configs():
    """make_shared_workload: the 1-D arrays the materialised Poisson config is made of (f3).  a, c and
    the real part of d are bit-identical to the materialised arrays; b agrees to rounding (the
    shared form subtracts sx + sz in one step); slices of a taller slab carry the bits of the full one."""
    import numpy as np
    w = ti.make_workload("cfg2_poisson", nz=3, nx=16, ny=32)
    for cplx in (False, True):
        s = ti.make_shared_workload("cfg2_poisson", cplx, nz=3, nx=16, ny=32)
        assert s.ncomp == (2 if cplx else 1) and s.pin00 and s.d.shape == (3, 32, 16)
        assert torch.equal(s.a_y, w.a[1, :, 5]) and torch.equal(s.c_y, w.c[2, :, 7])
        assert torch.equal(s.d.real if cplx else s.d, w.d)
        b = s.b0_y.view(1, -1, 1) - (s.sx.view(1, 1, -1) + s.sz.view(-1, 1, 1))
        b[0, 0, 0] = 1.0
        assert torch.allclose(b, w.b, rtol=1e-14, atol=0)
        assert s.d[0, 0, 0] == 0
        if cplx:
            assert float(s.d.imag.abs().max()) > 0 and not torch.equal(s.d.imag, s.d.real)
    full = ti.make_shared_workload("cfg2_poisson", True, nz=6, nx=16, ny=32)
    part = ti.make_shared_workload("cfg2_poisson", True, nz=2, nx=16, ny=32, k_offset=3)
    assert torch.equal(part.d, full.d[3:5]) and torch.equal(part.sz, full.sz[3:5]) and not part.pin00
    with pytest.raises(ValueError):
        ti.make_shared_workload("cfg1_tiny", False)
