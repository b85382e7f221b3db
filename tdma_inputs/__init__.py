"""Seeded synthetic inputs for the batched y-direction tridiagonal solve.

This module serves BOTH sides of the parity check (the CPU oracle under ``oracle/``
and the CUDA path under ``paper_2509_03933_b200/``) and therefore holds none of the
method's arithmetic: it only draws coefficients ``a, b, c`` (sub / main / super
diagonal) and right-hand sides ``d`` of the shapes and value
distributions of the BASELINE.json configs.  It imports neither side.

Layout (SURVEY.md notation): every array is a C-contiguous tensor of shape
``(nz, ny, nx)``, i.e. element (i, j, k) sits at ``i + nx*(j + ny*k)`` -- x fastest,
systems run along y (Fig. 1c).

Random numbers come from a counter-based generator (SplitMix64 finaliser applied to
``seed``/``stream``/linear cell index) written with integer tensor ops only, so the
uniform draws are bit-identical on CPU and on CUDA and for any z-chunking.  Normal
draws (Box-Muller) go through the device's log/cos and may differ in the last bit
between devices; a test always generates once and copies the same bits to both sides.

The five workload recipes:
  cfg 1  dominant_random      64^3,  P=4,  batch=all, seed 0
  cfg 2  poisson (tanh beta=2) 256^3, P=8
  cfg 3  poisson (uniform y)  1024^3, P=16, batch sweep 1..64
  cfg 4  adi_toeplitz (y sweep) 512^3, P=8
  cfg 5  dominant_random      2048x512x1024, P=64, batch sweep 1..128
These stand in for the flow-solver fields of the paper, which are not
available; nothing here is copied from a benchmark suite.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Dict, Optional, Tuple

import torch

__all__ = [
    "Workload", "CONFIGS", "config_spec", "make_workload", "uniform01", "normal01",
    "dominant_random", "poisson_wavenumber", "adi_toeplitz", "identity_system",
    "SharedWorkload", "poisson_shared", "make_shared_workload",
]

_MASK64 = (1 << 64) - 1
_GOLDEN = 0x9E3779B97F4A7C15
_MIX1 = 0xBF58476D1CE4E5B9
_MIX2 = 0x94D049BB133111EB


def _s64(v: int) -> int:
    """Two's-complement view of an unsigned 64-bit constant (torch has no uint64 math)."""
    v &= _MASK64
    return v - (1 << 64) if v >= (1 << 63) else v


def _lsr(z: torch.Tensor, n: int) -> torch.Tensor:
    """Logical shift right on int64 (torch's >> is arithmetic)."""
    return (z >> n) & ((1 << (64 - n)) - 1)


def _splitmix(idx: torch.Tensor, seed: int, stream: int) -> torch.Tensor:
    """SplitMix64 output for counter ``idx`` (int64 tensor), keyed by (seed, stream)."""
    key = (seed * _GOLDEN + (stream + 1) * _MIX1) & _MASK64
    z = idx * _s64(_GOLDEN) + _s64(key)
    z = (z ^ _lsr(z, 30)) * _s64(_MIX1)
    z = (z ^ _lsr(z, 27)) * _s64(_MIX2)
    return z ^ _lsr(z, 31)


def splitmix64_reference(counter: int, seed: int, stream: int) -> int:
    """Pure-Python big-int version of ``_splitmix`` (used by the tests as a pin)."""
    key = (seed * _GOLDEN + (stream + 1) * _MIX1) & _MASK64
    z = (counter * _GOLDEN + key) & _MASK64
    z = ((z ^ (z >> 30)) * _MIX1) & _MASK64
    z = ((z ^ (z >> 27)) * _MIX2) & _MASK64
    return z ^ (z >> 31)


def _cell_index(nx: int, ny: int, k0: int, k1: int, device) -> torch.Tensor:
    """Linear storage index i + nx*(j + ny*k) for slices k0..k1-1, shape (k1-k0, ny, nx)."""
    n = (k1 - k0) * ny * nx
    base = k0 * ny * nx
    return torch.arange(base, base + n, dtype=torch.int64, device=device).view(k1 - k0, ny, nx)


def uniform01(idx: torch.Tensor, seed: int, stream: int) -> torch.Tensor:
    """U[0,1) doubles with 53 random bits, one per entry of the int64 counter tensor."""
    return _lsr(_splitmix(idx, seed, stream), 11).to(torch.float64) * (2.0 ** -53)


def normal01(idx: torch.Tensor, seed: int, stream: int) -> torch.Tensor:
    """N(0,1) doubles by Box-Muller from two independent uniform streams."""
    u1 = 1.0 - uniform01(idx, seed, stream)            # (0,1]
    u2 = uniform01(idx, seed, stream + 1000)
    return torch.sqrt(-2.0 * torch.log(u1)) * torch.cos((2.0 * math.pi) * u2)


@dataclass
class Workload:
    """One synthetic slab: shapes, partition count P, batch (z-slices per pipeline stage)
    and the four input arrays, each of shape (nz, ny, nx)."""
    name: str
    nx: int
    ny: int
    nz: int
    P: int
    batch: int                      # 0 = all slices in one batch (BASELINE cfg 1 "batch=all")
    a: torch.Tensor
    b: torch.Tensor
    c: torch.Tensor
    d: torch.Tensor
    strictly_dominant: bool
    meta: Dict[str, float] = field(default_factory=dict)

    @property
    def cells(self) -> int:
        return self.nx * self.ny * self.nz


# name -> (kind, nx, ny, nz, P, batch, seed, extra)
CONFIGS: Dict[str, Tuple] = {
    "cfg1_tiny":     ("dominant_random", 64, 64, 64, 4, 0, 0, {}),
    "cfg2_poisson":  ("poisson", 256, 256, 256, 8, 32, 1, {"beta": 2.0}),
    "cfg3_weak":     ("poisson", 1024, 1024, 1024, 16, 32, 2, {"beta": None}),
    "cfg4_adi_y":    ("adi_toeplitz", 512, 512, 512, 8, 32, 3, {}),
    "cfg5_stress":   ("dominant_random", 2048, 512, 1024, 64, 16, 4, {}),
}


def config_spec(name: str) -> Dict:
    kind, nx, ny, nz, P, batch, seed, extra = CONFIGS[name]
    return dict(kind=kind, nx=nx, ny=ny, nz=nz, P=P, batch=batch, seed=seed, **extra)


def _chunks(nz: int, ny: int, nx: int, target_cells: int = 1 << 24):
    step = max(1, target_cells // (ny * nx))
    k = 0
    while k < nz:
        yield k, min(nz, k + step)
        k += step


def dominant_random(nx: int, ny: int, nz: int, seed: int, device="cpu",
                    k_offset: int = 0, nz_total: Optional[int] = None):
    """BASELINE cfg 1/5: a,c ~ U(-1,1); b = 2+|a|+|c|+U(0,1); d ~ U(-1,1), drawn per cell.

    ``k_offset``/``nz_total`` let a caller generate only slices [k_offset, k_offset+nz)
    of a taller slab with the same bits the full slab would have (counter = global cell
    index)."""
    a = torch.empty((nz, ny, nx), dtype=torch.float64, device=device)
    b, c, d = torch.empty_like(a), torch.empty_like(a), torch.empty_like(a)
    for k0, k1 in _chunks(nz, ny, nx):
        idx = _cell_index(nx, ny, k_offset + k0, k_offset + k1, device)
        ua = 2.0 * uniform01(idx, seed, 0) - 1.0
        uc = 2.0 * uniform01(idx, seed, 1) - 1.0
        a[k0:k1] = ua
        c[k0:k1] = uc
        b[k0:k1] = 2.0 + ua.abs() + uc.abs() + uniform01(idx, seed, 2)
        d[k0:k1] = 2.0 * uniform01(idx, seed, 3) - 1.0
        del idx, ua, uc
    return a, b, c, d


def poisson_y_coefficients(ny: int, beta: Optional[float]):
    """1-D second-order finite-difference weights on a (stretched) cell-centred y grid.

    Faces y_f(q) = tanh(beta*xi_q)/tanh(beta), xi_q = -1 + 2q/ny, q = 0..ny  (beta None:
    uniform, y_f = xi).  h_j = y_f(j+1)-y_f(j); centres y_c(j) = (y_f(j)+y_f(j+1))/2;
    a_j = 1/(h_j*(y_c(j)-y_c(j-1))), c_j = 1/(h_j*(y_c(j+1)-y_c(j))); Neumann walls by
    ghost-cell folding: a_0 = 0, c_{ny-1} = 0.
    Returns float64 CPU tensors (a_y, c_y) of length ny."""
    q = torch.arange(ny + 1, dtype=torch.float64)
    xi = -1.0 + 2.0 * q / ny
    yf = xi if beta is None else torch.tanh(beta * xi) / math.tanh(beta)
    h = yf[1:] - yf[:-1]
    yc = 0.5 * (yf[1:] + yf[:-1])
    dyc = yc[1:] - yc[:-1]                       # length ny-1, dyc[j] = yc(j+1)-yc(j)
    a_y = torch.zeros(ny, dtype=torch.float64)
    c_y = torch.zeros(ny, dtype=torch.float64)
    a_y[1:] = 1.0 / (h[1:] * dyc)
    c_y[:-1] = 1.0 / (h[:-1] * dyc)
    return a_y, c_y


def poisson_wavenumber(nx: int, ny: int, nz: int, seed: int, beta: Optional[float],
                       device="cpu", Lx: float = 2.0 * math.pi, Lz: float = 2.0 * math.pi,
                       k_offset: int = 0, nz_total: Optional[int] = None):
    """BASELINE cfg 2/3: FFT-reduced Poisson lines (d^2/dy^2 - kx^2 - kz^2) Phi = Q
    (PAPER.md:286): b_j = -(a_j+c_j) - kx^2 - kz^2 with modified wavenumbers
    kx = 2 sin(pi i/nx)/dx, kz = 2 sin(pi k/nz)/dz; mode (0,0) pinned by x_0 = 0
    (row 0 := b=1, c=0, d=0); d ~ N(0,1).  a, c, b are materialised as full 3-D arrays
    (the API contract is 40 B/cell)."""
    nzt = nz if nz_total is None else nz_total
    a_y, c_y = poisson_y_coefficients(ny, beta)
    a_y, c_y = a_y.to(device), c_y.to(device)
    dx, dz = Lx / nx, Lz / nzt
    i = torch.arange(nx, dtype=torch.float64, device=device)
    k = torch.arange(k_offset, k_offset + nz, dtype=torch.float64, device=device)
    kx2 = (2.0 * torch.sin(math.pi * i / nx) / dx) ** 2
    kz2 = (2.0 * torch.sin(math.pi * k / nzt) / dz) ** 2
    a = a_y.view(1, ny, 1).expand(nz, ny, nx).contiguous()
    c = c_y.view(1, ny, 1).expand(nz, ny, nx).contiguous()
    b = torch.empty((nz, ny, nx), dtype=torch.float64, device=device)
    d = torch.empty_like(b)
    diag_y = -(a_y + c_y).view(1, ny, 1)
    for k0, k1 in _chunks(nz, ny, nx):
        b[k0:k1] = diag_y - kx2.view(1, 1, nx) - kz2[k0:k1].view(-1, 1, 1)
        idx = _cell_index(nx, ny, k_offset + k0, k_offset + k1, device)
        d[k0:k1] = normal01(idx, seed, 0)
        del idx
    if k_offset == 0:                             # (i,k) = (0,0): pin x_0 = 0
        b[0, 0, 0] = 1.0
        c[0, 0, 0] = 0.0
        d[0, 0, 0] = 0.0
    return a, b, c, d


@dataclass
class SharedWorkload:
    """Shared-coefficient form of a Poisson config: line (i,k) has a = a_y,
    c = c_y, b = b0_y - (sx[i] + sz[k]); d real or complex (nz, ny, nx)."""
    name: str
    nx: int
    ny: int
    nz: int
    a_y: torch.Tensor
    b0_y: torch.Tensor
    c_y: torch.Tensor
    sx: torch.Tensor
    sz: torch.Tensor
    d: torch.Tensor
    pin00: bool
    meta: Dict[str, float] = field(default_factory=dict)

    @property
    def cells(self) -> int:
        return self.nx * self.ny * self.nz

    @property
    def ncomp(self) -> int:
        return 2 if self.d.is_complex() else 1


def poisson_shared(nx: int, ny: int, nz: int, seed: int, beta: Optional[float], cplx: bool, device="cpu",
                   Lx: float = 2.0 * math.pi, Lz: float = 2.0 * math.pi, k_offset: int = 0,
                   nz_total: Optional[int] = None):
    """The coefficients of ``poisson_wavenumber`` as the 1-D arrays they are made of (PAPER.md:286,
    318): a_y, c_y, b0_y = -(a_y + c_y), sx = kx^2, sz = kz^2; d ~ N(0,1) per component (complex
    fields: PAPER.md:377; re uses stream 0 -- the bits of the real config -- and im stream 1);
    mode (0,0) pinned (pin00) with d_0 = 0."""
    nzt = nz if nz_total is None else nz_total
    a_y, c_y = poisson_y_coefficients(ny, beta)
    a_y, c_y = a_y.to(device), c_y.to(device)
    dx, dz = Lx / nx, Lz / nzt
    i = torch.arange(nx, dtype=torch.float64, device=device)
    k = torch.arange(k_offset, k_offset + nz, dtype=torch.float64, device=device)
    sx = (2.0 * torch.sin(math.pi * i / nx) / dx) ** 2
    sz = (2.0 * torch.sin(math.pi * k / nzt) / dz) ** 2
    d = torch.empty((nz, ny, nx), dtype=torch.complex128 if cplx else torch.float64, device=device)
    dv = torch.view_as_real(d) if cplx else d.unsqueeze(-1)
    for k0, k1 in _chunks(nz, ny, nx):
        idx = _cell_index(nx, ny, k_offset + k0, k_offset + k1, device)
        for q in range(2 if cplx else 1):
            dv[k0:k1, :, :, q] = normal01(idx, seed, q)
        del idx
    if k_offset == 0:
        d[0, 0, 0] = 0.0
    return a_y, -(a_y + c_y), c_y, sx, sz, d


def make_shared_workload(name: str, cplx: bool, device="cpu", nz: Optional[int] = None, nx: Optional[int] = None,
                         ny: Optional[int] = None, k_offset: int = 0) -> SharedWorkload:
    """Shared-coefficient form of a ``poisson`` config (cfg2_poisson, cfg3_weak); ``nz`` / ``k_offset``
    restrict generation to a z-range with the bits of the full slab."""
    spec = config_spec(name)
    if spec["kind"] != "poisson":
        raise ValueError("shared-coefficient workloads are defined for the Poisson configs")
    fnx = spec["nx"] if nx is None else nx
    fny = spec["ny"] if ny is None else ny
    gnz = spec["nz"] if nz is None else nz
    a_y, b0_y, c_y, sx, sz, d = poisson_shared(fnx, fny, gnz, spec["seed"], spec["beta"], cplx, device,
                                               k_offset=k_offset, nz_total=spec["nz"])
    return SharedWorkload(name + ("_shared_c128" if cplx else "_shared_f64"), fnx, fny, gnz, a_y, b0_y, c_y, sx, sz, d,
                          pin00=(k_offset == 0), meta={"seed": spec["seed"], "k_offset": k_offset})


def adi_alpha(seed: int) -> float:
    """alpha = nu*dt/h^2 ~ U(0.1, 10), one scalar per run (BASELINE cfg 4)."""
    u = uniform01(torch.zeros(1, dtype=torch.int64), seed, 7).item()
    return 0.1 + 9.9 * u


def adi_toeplitz(nx: int, ny: int, nz: int, seed: int, device="cpu", alpha: Optional[float] = None,
                 k_offset: int = 0, nz_total: Optional[int] = None):
    """BASELINE cfg 4, y sweep: a = c = -alpha, b = 1+2 alpha (Dirichlet in y), d ~ U(-1,1)
    ((1 - A_y) is diagonally dominant with small off-diagonals)."""
    al = adi_alpha(seed) if alpha is None else float(alpha)
    a = torch.full((nz, ny, nx), -al, dtype=torch.float64, device=device)
    c = a.clone()
    b = torch.full((nz, ny, nx), 1.0 + 2.0 * al, dtype=torch.float64, device=device)
    d = torch.empty_like(a)
    for k0, k1 in _chunks(nz, ny, nx):
        idx = _cell_index(nx, ny, k_offset + k0, k_offset + k1, device)
        d[k0:k1] = 2.0 * uniform01(idx, seed, 3) - 1.0
        del idx
    return a, b, c, d, al


def identity_system(nx: int, ny: int, nz: int, seed: int, device="cpu", diagonal_only: bool = False):
    """Degenerate plumbing cases: identity (x = d) or diagonal (x = d/b)."""
    idx = _cell_index(nx, ny, 0, nz, device)
    a = torch.zeros((nz, ny, nx), dtype=torch.float64, device=device)
    c = torch.zeros_like(a)
    b = (1.0 + uniform01(idx, seed, 2)) if diagonal_only else torch.ones_like(a)
    d = 2.0 * uniform01(idx, seed, 3) - 1.0
    return a, b, c, d


def make_workload(name: str, device="cpu", nz: Optional[int] = None, nx: Optional[int] = None,
                  ny: Optional[int] = None, P: Optional[int] = None, batch: Optional[int] = None,
                  k_offset: int = 0) -> Workload:
    """Build a BASELINE config by name.  ``nz`` (and ``k_offset``) restrict generation to a
    z-range of the full slab, with the same values those slices have in the full slab --
    this is how the bounded oracle samples of the 1e9-cell configs are produced."""
    spec = config_spec(name)
    kind = spec["kind"]
    fnx = spec["nx"] if nx is None else nx
    fny = spec["ny"] if ny is None else ny
    full_nz = spec["nz"]
    gnz = full_nz if nz is None else nz
    fP = spec["P"] if P is None else P
    fb = spec["batch"] if batch is None else batch
    seed = spec["seed"]
    meta: Dict[str, float] = {"seed": seed, "k_offset": k_offset, "nz_total": full_nz}
    if kind == "dominant_random":
        a, b, c, d = dominant_random(fnx, fny, gnz, seed, device, k_offset, full_nz)
        dom = True
    elif kind == "poisson":
        a, b, c, d = poisson_wavenumber(fnx, fny, gnz, seed, spec["beta"], device,
                                        k_offset=k_offset, nz_total=full_nz)
        meta["beta"] = -1.0 if spec["beta"] is None else spec["beta"]
        dom = False                                # weakly dominant near (kx,kz) -> 0
    elif kind == "adi_toeplitz":
        a, b, c, d, al = adi_toeplitz(fnx, fny, gnz, seed, device, k_offset=k_offset,
                                      nz_total=full_nz)
        meta["alpha"] = al
        dom = True
    else:
        raise ValueError(kind)
    return Workload(name, fnx, fny, gnz, fP, fb, a, b, c, d, dom, meta)
