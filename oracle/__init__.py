"""ORACLE -- TEST INFRASTRUCTURE ONLY (never imported by the product package).

Plain CPU definition of the batched y-direction tridiagonal solve, used by ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs.

  * ``solve_y(a, b, c, d, precision="f64"|"ld")``  -- textbook Thomas per line
    (problem statement PAPER.md:127-131, 210), implemented in
    ``thomas_oracle.c`` (gcc, fp-contraction off so no FMA sneaks in).
  * ``residual_y`` / ``apply_y``                   -- long-double residual and d = A x.
  * ``solve_y_shared``                             -- SURVEY 8(f) f3: 1-D coefficients shared by all
    lines, diagonal shifted per line, real or complex right-hand sides.
  * ``reduced_rows_y`` / ``solve_y_pdd``           -- SURVEY 8(f) f4: the 2P-row reduced system by its
    definition (Schur complement), and the PDD approximation (Sun 1995) step by step.
  * ``thomas_line``                                -- the same recurrence as a pure-Python loop
    for one small line (brute-force cross-checks).

Parity status: pinned (tests/test_oracle_pins.py): dense LAPACK solve n<=32, banded LAPACK,
manufactured solutions, Toeplitz closed forms (eigen-form and Green's function), identity /
diagonal / n=1,2 degenerate cases, long-double vs fp64 agreement.  The paper prints no worked
numerical example (Figs. 3-4 are images), so there is no paper-value pin.

Nothing here imports or links anything from ``paper_2509_03933_b200``.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "thomas_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile thomas_oracle.c -> liboracle.so (gcc -O2 -fopenmp -ffp-contract=off)."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    tmp = _LIB + ".tmp.%d" % os.getpid()
    cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
           "-o", tmp, _SRC, "-lm"]
    subprocess.run(cmd, check=True, capture_output=True, text=True)
    os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        lib.oracle_solve_y.argtypes = [ctypes.c_int] * 3 + [dp] * 5 + [ctypes.c_int]
        lib.oracle_solve_y.restype = ctypes.c_int
        lib.oracle_residual_y.argtypes = [ctypes.c_int] * 3 + [dp] * 9
        lib.oracle_residual_y.restype = ctypes.c_int
        lib.oracle_apply_y.argtypes = [ctypes.c_int] * 3 + [dp] * 5
        lib.oracle_apply_y.restype = ctypes.c_int
        lib.oracle_solve_y_shared.argtypes = [ctypes.c_int] * 4 + [dp] * 5 + [ctypes.c_int] + [dp] * 2 + [ctypes.c_int]
        lib.oracle_solve_y_shared.restype = ctypes.c_int
        lib.oracle_max_threads.restype = ctypes.c_int
        lib.oracle_set_threads.argtypes = [ctypes.c_int]
        _lib = lib
    return _lib


def _as3(arr) -> np.ndarray:
    out = np.ascontiguousarray(np.asarray(arr, dtype=np.float64))
    if out.ndim != 3:
        raise ValueError("expected an array of shape (nz, ny, nx)")
    return out


def _ptr(arr: np.ndarray):
    return arr.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def max_threads() -> int:
    return int(_load().oracle_max_threads())


def set_threads(n: int) -> None:
    _load().oracle_set_threads(int(n))


def solve_y(a, b, c, d, precision: str = "f64") -> np.ndarray:
    """x with A x = d for every y-line; arrays of shape (nz, ny, nx), x fastest."""
    a, b, c, d = map(_as3, (a, b, c, d))
    if not (a.shape == b.shape == c.shape == d.shape):
        raise ValueError("a, b, c, d must have the same shape")
    nz, ny, nx = a.shape
    x = np.empty_like(d)
    use_ld = {"f64": 0, "ld": 1}[precision]
    rc = _load().oracle_solve_y(nx, ny, nz, _ptr(a), _ptr(b), _ptr(c), _ptr(d), _ptr(x), use_ld)
    if rc != 0:
        raise RuntimeError("oracle_solve_y failed (%d)" % rc)
    return x


def residual_y(a, b, c, d, x) -> Tuple[np.ndarray, np.ndarray, np.ndarray, np.ndarray]:
    """Per line (shape (nz, nx)): ||Ax-d||_inf, ||d||_inf, ||x||_inf, ||A||_inf; long double."""
    a, b, c, d, x = map(_as3, (a, b, c, d, x))
    nz, ny, nx = a.shape
    outs = [np.empty((nz, nx), dtype=np.float64) for _ in range(4)]
    rc = _load().oracle_residual_y(nx, ny, nz, _ptr(a), _ptr(b), _ptr(c), _ptr(d), _ptr(x),
                                   *[_ptr(o) for o in outs])
    if rc != 0:
        raise RuntimeError("oracle_residual_y failed (%d)" % rc)
    return tuple(outs)


def apply_y(a, b, c, x) -> np.ndarray:
    """d = A x per line, accumulated in long double and rounded once."""
    a, b, c, x = map(_as3, (a, b, c, x))
    nz, ny, nx = a.shape
    d = np.empty_like(x)
    rc = _load().oracle_apply_y(nx, ny, nz, _ptr(a), _ptr(b), _ptr(c), _ptr(x), _ptr(d))
    if rc != 0:
        raise RuntimeError("oracle_apply_y failed (%d)" % rc)
    return d


def thomas_line(a: Sequence[float], b: Sequence[float], c: Sequence[float],
                d: Sequence[float]) -> list:
    """Thomas algorithm for ONE line as a pure-Python loop; tiny inputs only."""
    n = len(b)
    cp = [0.0] * n
    dp = [0.0] * n
    cp[0] = (c[0] / b[0]) if n > 1 else 0.0
    dp[0] = d[0] / b[0]
    for j in range(1, n):
        den = b[j] - a[j] * cp[j - 1]
        cp[j] = (c[j] / den) if j < n - 1 else 0.0
        dp[j] = (d[j] - a[j] * dp[j - 1]) / den
    x = [0.0] * n
    x[n - 1] = dp[n - 1]
    for j in range(n - 2, -1, -1):
        x[j] = dp[j] - cp[j] * x[j + 1]
    return x


def normwise_error(x: np.ndarray, x_ref: np.ndarray) -> np.ndarray:
    """Per-line E = ||x - x_ref||_inf / ||x_ref||_inf, shape (nz, nx).
    Lines whose reference is identically zero report the absolute error."""
    x, x_ref = _as3(x), _as3(x_ref)
    num = np.max(np.abs(x - x_ref), axis=1)
    den = np.max(np.abs(x_ref), axis=1)
    return np.where(den > 0, num / np.where(den > 0, den, 1.0), num)


# ---------------------------------------------------------------------------------------------
# sweeps along z and cyclic (periodic) lines (BASELINE cfg 4)
# ---------------------------------------------------------------------------------------------
def solve_cyclic_y(a, b, c, d, precision: str = "f64") -> np.ndarray:
    """Cyclic tridiagonal lines along y: row 0 couples to row n-1 through a_0 and row n-1 to row 0
    through c_{n-1}.  Sherman-Morrison on top of the Thomas oracle, exactly as written in
    SURVEY.md 8(f) f1:  gamma = -b_0;  b'_0 = b_0 - gamma;  b'_{n-1} = b_{n-1} - c_{n-1} a_0/gamma;
    A' y = d;  A' q = u,  u = (gamma, 0, ..., 0, c_{n-1})^T;
    x = y - q (y_0 + a_0 y_{n-1}/gamma) / (1 + q_0 + a_0 q_{n-1}/gamma).
    Pinned in tests/test_oracle_pins.py against dense LAPACK solves of the full cyclic matrix and
    the circulant closed form x = IFFT(FFT(d)/lambda)."""
    a, b, c, d = map(_as3, (a, b, c, d))
    n = a.shape[1]
    if n < 3:
        raise ValueError("cyclic lines need n >= 3")
    a0, cn = a[:, 0, :], c[:, n - 1, :]
    gamma = -b[:, 0, :]
    bp = b.copy()
    bp[:, 0, :] = b[:, 0, :] - gamma
    bp[:, n - 1, :] = b[:, n - 1, :] - cn * a0 / gamma
    u = np.zeros_like(d)
    u[:, 0, :] = gamma
    u[:, n - 1, :] = cn
    y = solve_y(a, bp, c, d, precision).astype(np.longdouble)
    q = solve_y(a, bp, c, u, precision).astype(np.longdouble)
    g = gamma.astype(np.longdouble)
    fac = (y[:, 0, :] + a0 * y[:, n - 1, :] / g) / (1.0 + q[:, 0, :] + a0 * q[:, n - 1, :] / g)
    return np.asarray(y - q * fac[:, None, :], dtype=np.float64)


def solve_axis(a, b, c, d, axis: str = "y", periodic: bool = False, precision: str = "f64") -> np.ndarray:
    """Lines along x, y or z of (nz, ny, nx) arrays: an x / z sweep is the y sweep of the arrays
    with the solve axis exchanged with y."""
    perm = {"y": None, "z": (1, 0, 2), "x": (0, 2, 1)}[axis]     # brings the solve axis to position 1
    arrs = [_as3(t) for t in (a, b, c, d)]
    if perm:
        arrs = [np.ascontiguousarray(t.transpose(perm)) for t in arrs]
    x = (solve_cyclic_y if periodic else solve_y)(*arrs, precision)
    return np.ascontiguousarray(x.transpose(perm)) if perm else x


# ---------------------------------------------------------------------------------------------
# shared coefficients, complex right-hand sides
# ---------------------------------------------------------------------------------------------
def solve_y_shared(a_y, b0_y, c_y, sx, sz, d, pin00: bool = False, precision: str = "f64") -> np.ndarray:
    """Lines along y whose matrix is given by 1-D arrays: a_j = a_y[j], c_j = c_y[j],
    b_j = b0_y[j] - (sx[i] + sz[k]) for line (i, k) ((d2/dy2 - k_l - k_m) Phi = Q;
    PAPER.md:318: the matrix depends solely on grid spacing).  ``d`` has shape (nz, ny, nx), real
    or complex (complex-valued data, real coefficients: each of re / im is a
    right-hand side of the same matrix).  pin00: row 0 of line (0, 0) is b = 1, c = 0.
    Plain Thomas per line and component (thomas_oracle.c: oracle_solve_y_shared).
    Pinned in tests/test_oracle_pins.py: bit-equal to ``solve_y`` on the materialised arrays,
    dense LAPACK solve of the complex system for n <= 32, Toeplitz eigen-form with a shift."""
    a_y, b0_y, c_y, sx, sz = [np.ascontiguousarray(np.asarray(t, dtype=np.float64)) for t in (a_y, b0_y, c_y, sx, sz)]
    d = np.asarray(d)
    cplx = np.iscomplexobj(d)
    d = np.ascontiguousarray(d, dtype=np.complex128 if cplx else np.float64)
    if d.ndim != 3:
        raise ValueError("expected d of shape (nz, ny, nx)")
    nz, ny, nx = d.shape
    if a_y.shape != (ny,) or b0_y.shape != (ny,) or c_y.shape != (ny,) or sx.shape != (nx,) or sz.shape != (nz,):
        raise ValueError("coefficient arrays must have lengths ny, ny, ny, nx, nz")
    x = np.empty_like(d)
    dv, xv = d.view(np.float64), x.view(np.float64)
    rc = _load().oracle_solve_y_shared(nx, ny, nz, 2 if cplx else 1, _ptr(a_y), _ptr(b0_y), _ptr(c_y), _ptr(sx),
                                       _ptr(sz), 1 if pin00 else 0, _ptr(dv), _ptr(xv),
                                       {"f64": 0, "ld": 1}[precision])
    if rc != 0:
        raise RuntimeError("oracle_solve_y_shared failed (%d)" % rc)
    return x


# ---------------------------------------------------------------------------------------------
# SURVEY 8(f) f4, PDD variant ("Parallel Diagonally Dominant (PDD) method [37] ...
# designed for diagonally dominant TDM systems"; SURVEY: "PDD = drop the reduced solve's far
# coupling when spikes decay")
# ---------------------------------------------------------------------------------------------
def reduced_rows_y(a, b, c, d, P: int, precision: str = "f64"):
    """The 2P-row reduced system of the P-partition split, BY DEFINITION (Schur complement of the
    interior rows of every partition), unit diagonal:
        row 2p  :  fa x_last(p-1) + x_first(p) + fc x_last(p)  = fd
        row 2p+1:  pa x_first(p) + x_last(p)  + pc x_first(p+1) = pd
    Returned as arrays of shape (P, nz, nx): fa, fc, fd, pa, pc, pd.  The interior solves are plain
    Thomas solves (solve_y) of rows 1 .. m-2 of a partition with three right-hand sides."""
    a, b, c, d = map(_as3, (a, b, c, d))
    nz, ny, nx = a.shape
    if ny % P or ny // P < 2:
        raise ValueError("ny must split into P partitions of >= 2 rows")
    m = ny // P
    out = [np.zeros((P, nz, nx)) for _ in range(6)]
    for p in range(P):
        r0 = p * m
        A, B, C, D = [np.array(t[:, r0:r0 + m, :], dtype=np.float64) for t in (a, b, c, d)]
        if p == 0:
            A[:, 0, :] = 0.0
        if p == P - 1:
            C[:, m - 1, :] = 0.0
        if m == 2:
            g0 = gl = u0 = ul = v0 = vl = None
            out[0][p], out[1][p], out[2][p] = A[:, 0] / B[:, 0], C[:, 0] / B[:, 0], D[:, 0] / B[:, 0]
            out[3][p], out[4][p], out[5][p] = A[:, 1] / B[:, 1], C[:, 1] / B[:, 1], D[:, 1] / B[:, 1]
            continue
        ai, bi, ci = [np.ascontiguousarray(t[:, 1:m - 1, :]) for t in (A, B, C)]
        ef, el = np.zeros_like(bi), np.zeros_like(bi)
        ef[:, 0, :] = A[:, 1, :]                  # a_1 x_0 moved to the right-hand side
        el[:, -1, :] = C[:, m - 2, :]             # c_{m-2} x_{m-1}
        g = solve_y(ai, bi, ci, np.ascontiguousarray(D[:, 1:m - 1, :]), precision)
        u = solve_y(ai, bi, ci, ef, precision)
        v = solve_y(ai, bi, ci, el, precision)    # x_int = g - u x_0 - v x_{m-1}
        diag = B[:, 0] - C[:, 0] * u[:, 0]
        out[0][p], out[1][p], out[2][p] = A[:, 0] / diag, -C[:, 0] * v[:, 0] / diag, (D[:, 0] - C[:, 0] * g[:, 0]) / diag
        diag = B[:, m - 1] - A[:, m - 1] * v[:, -1]
        out[3][p], out[4][p] = -A[:, m - 1] * u[:, -1] / diag, C[:, m - 1] / diag
        out[5][p] = (D[:, m - 1] - A[:, m - 1] * g[:, -1]) / diag
    return tuple(out)


def solve_y_pdd(a, b, c, d, P: int, precision: str = "f64") -> np.ndarray:
    """The Parallel Diagonally Dominant algorithm (Sun, Parallel Computing 21 (1995), the paper's
    [37]), step by step, for the P-partition split of every line (m = ny / P rows
    per partition, block p = rows p m .. p m + m - 1, A_p its tridiagonal block):
      1. three Thomas solves per block:  A_p xt = d_p,   A_p v = a_first e_0,   A_p w = c_last e_{m-1}
         (a_first = the block's coupling to the row above it, c_last = to the row below it; the
         spikes v, w decay away from the block end they start at);
      2. the exact solution is  x_p = xt - v y_l(p-1) - w y_f(p+1)  with the interface unknowns
         y_l(p) = x_last(p), y_f(p) = x_first(p); PDD DROPS the far ends of the spikes, w_0 and
         v_{m-1}, which leaves one 2 x 2 system per interface:
              y_l(p) + w^p_{m-1} y_f(p+1) = xt^p_{m-1} ,    v^{p+1}_0 y_l(p) + y_f(p+1) = xt^{p+1}_0 ;
      3. x_p = xt - v y_l(p-1) - w y_f(p+1)  with those y (y_l(-1) = y_f(P) = 0).
    Exact when the blocks do not couple; otherwise the error is of the order of the dropped
    entries, which decay geometrically with m for strictly dominant systems (pinned in
    tests/test_oracle_pins.py)."""
    a, b, c, d = map(_as3, (a, b, c, d))
    nz, ny, nx = a.shape
    if ny % P or ny // P < 2:
        raise ValueError("ny must split into P partitions of >= 2 rows")
    m = ny // P
    xt, v, w = np.empty_like(d), np.zeros_like(d), np.zeros_like(d)
    for p in range(P):
        r = slice(p * m, (p + 1) * m)
        blk = [np.ascontiguousarray(t[:, r, :]) for t in (a, b, c)]
        xt[:, r, :] = solve_y(*blk, np.ascontiguousarray(d[:, r, :]), precision)
        if p > 0:
            e = np.zeros((nz, m, nx)); e[:, 0, :] = a[:, p * m, :]
            v[:, r, :] = solve_y(*blk, e, precision)
        if p < P - 1:
            e = np.zeros((nz, m, nx)); e[:, m - 1, :] = c[:, p * m + m - 1, :]
            w[:, r, :] = solve_y(*blk, e, precision)
    yl = np.zeros((P + 1, nz, nx)); yf = np.zeros((P + 1, nz, nx))     # yl[p] = y_l(p-1), yf[p] = y_f(p)
    for p in range(P - 1):
        wl, v0 = w[:, p * m + m - 1, :], v[:, (p + 1) * m, :]
        tl, t0 = xt[:, p * m + m - 1, :], xt[:, (p + 1) * m, :]
        det = 1.0 - wl * v0
        yl[p + 1] = (tl - wl * t0) / det
        yf[p + 1] = (t0 - v0 * tl) / det
    x = np.empty_like(d)
    for p in range(P):
        r = slice(p * m, (p + 1) * m)
        y_prev = yl[p][:, None, :]
        y_next = (yf[p + 1] if p < P - 1 else np.zeros((nz, nx)))[:, None, :]
        x[:, r, :] = xt[:, r, :] - v[:, r, :] * y_prev - w[:, r, :] * y_next
    return x
