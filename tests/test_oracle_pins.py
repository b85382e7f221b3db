"""Pins for the CPU oracle: the oracle is checked against things
other than itself before any CUDA result is compared with it.

  P1  dense brute force: Gaussian elimination with partial pivoting in long double written out
      here, and LAPACK dgesv (np.linalg.solve), n <= 32, NON-symmetric matrices (a != c) so a
      transposed operand fails
  P1b banded LAPACK (scipy.linalg.solve_banded) on Poisson-type and random lines up to n = 256
  P2  manufactured solutions: choose x*, form d = A x* with numpy long double, recover x*
  P3  residual ||Ax-d||_inf (evaluated here independently of the oracle's own evaluator)
  P4  closed forms of the constant-coefficient Toeplitz system a=c=-alpha, b=1+2alpha:
      eigen-form (sine modes) and Green's function; plus the exact rational inverse of the
      second-difference matrix tridiag(-1,2,-1) from tests/golden/second_difference_inverse.txt
  P7  degenerate cases: identity, diagonal, n = 1, n = 2, nx = 1, nz = 1, ignored a_0 / c_{n-1}
No paper-printed worked example exists (Figs. 3-4 are images).
"""
import math
import os

import numpy as np
import pytest
import scipy.linalg

import oracle

HERE = os.path.dirname(os.path.abspath(__file__))
LD = np.longdouble
PI_LD = np.longdouble("3.14159265358979323846264338327950288")


# ----------------------------------------------------------------------------------------------
# helpers written independently of oracle/
# ----------------------------------------------------------------------------------------------
def dense_from_line(a, b, c):
    n = len(b)
    A = np.zeros((n, n), dtype=LD)
    for j in range(n):
        A[j, j] = b[j]
        if j > 0:
            A[j, j - 1] = a[j]
        if j < n - 1:
            A[j, j + 1] = c[j]
    return A


def gauss_partial_pivot_ld(A, d):
    """Textbook Gaussian elimination with partial pivoting, long double."""
    A = np.array(A, dtype=LD)
    y = np.array(d, dtype=LD)
    n = len(y)
    for col in range(n):
        piv = col + int(np.argmax(np.abs(A[col:, col])))
        if piv != col:
            A[[col, piv]] = A[[piv, col]]
            y[[col, piv]] = y[[piv, col]]
        for row in range(col + 1, n):
            f = A[row, col] / A[col, col]
            if f != 0:
                A[row, col:] -= f * A[col, col:]
                y[row] -= f * y[col]
    x = np.zeros(n, dtype=LD)
    for row in range(n - 1, -1, -1):
        x[row] = (y[row] - np.dot(A[row, row + 1:], x[row + 1:])) / A[row, row]
    return x


def random_lines(rng, nz, ny, nx, dominant=True):
    a = rng.uniform(-1, 1, (nz, ny, nx))
    c = rng.uniform(-1, 1, (nz, ny, nx))
    if dominant:
        b = 2.0 + np.abs(a) + np.abs(c) + rng.uniform(0, 1, (nz, ny, nx))
        b *= rng.choice([-1.0, 1.0], (nz, 1, nx))          # both signs of the diagonal
    else:
        b = rng.uniform(2.5, 4.0, (nz, ny, nx))
    d = rng.uniform(-1, 1, (nz, ny, nx))
    return a, b, c, d


def apply_ld(a, b, c, x):
    """d = A x along axis 1 in numpy long double (a_0, c_{n-1} ignored)."""
    a, b, c, x = (np.asarray(v, dtype=LD) for v in (a, b, c, x))
    out = b * x
    out[:, 1:, :] += a[:, 1:, :] * x[:, :-1, :]
    out[:, :-1, :] += c[:, :-1, :] * x[:, 1:, :]
    return out


def rel_inf(x, ref):
    ref = np.asarray(ref, dtype=np.float64)
    return float(np.max(np.abs(np.asarray(x, dtype=np.float64) - ref)) / np.max(np.abs(ref)))


# ----------------------------------------------------------------------------------------------
# P1 dense brute force
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n", [1, 2, 3, 5, 8, 16, 31, 32])
@pytest.mark.parametrize("precision", ["f64", "ld"])
def test_p1_dense_gauss_long_double(n, precision):
    rng = np.random.default_rng(100 + n)
    nz, nx = 2, 3
    a, b, c, d = random_lines(rng, nz, n, nx)
    x = oracle.solve_y(a, b, c, d, precision)
    for k in range(nz):
        for i in range(nx):
            A = dense_from_line(a[k, :, i], b[k, :, i], c[k, :, i])
            ref = gauss_partial_pivot_ld(A, d[k, :, i])
            assert rel_inf(x[k, :, i], ref) <= 1e-14


@pytest.mark.parametrize("n", [4, 17, 32])
def test_p1_dense_lapack(n):
    rng = np.random.default_rng(7 + n)
    a, b, c, d = random_lines(rng, 3, n, 4, dominant=False)      # not strictly dominant either
    x = oracle.solve_y(a, b, c, d)
    for k in range(3):
        for i in range(4):
            A = dense_from_line(a[k, :, i], b[k, :, i], c[k, :, i]).astype(np.float64)
            ref = np.linalg.solve(A, d[k, :, i])
            assert rel_inf(x[k, :, i], ref) <= 5e-13


def test_p1_pure_python_loop_matches_c():
    rng = np.random.default_rng(3)
    a, b, c, d = random_lines(rng, 1, 24, 2)
    x = oracle.solve_y(a, b, c, d)
    for i in range(2):
        ref = oracle.thomas_line(list(a[0, :, i]), list(b[0, :, i]), list(c[0, :, i]), list(d[0, :, i]))
        # same recurrence, same precision, no FMA contraction on either side: bit-identical
        assert np.array_equal(x[0, :, i], np.array(ref))


def test_p1b_banded_lapack_poisson_lines():
    """Poisson-type line: stretched-grid weights, b = -(a+c) - k^2 (weakly dominant)."""
    import tdma_inputs
    ny = 256
    a_y, c_y = tdma_inputs.poisson_y_coefficients(ny, 2.0)
    a_y, c_y = a_y.numpy(), c_y.numpy()
    rng = np.random.default_rng(11)
    k2 = np.array([0.5, 3.0, 40.0, 1.0e4])
    nx = len(k2)
    a = np.broadcast_to(a_y[None, :, None], (1, ny, nx)).copy()
    c = np.broadcast_to(c_y[None, :, None], (1, ny, nx)).copy()
    b = -(a + c) - k2[None, None, :]
    d = rng.standard_normal((1, ny, nx))
    x = oracle.solve_y(a, b, c, d)
    xl = oracle.solve_y(a, b, c, d, "ld")
    for i in range(nx):
        ab = np.zeros((3, ny))
        ab[0, 1:] = c[0, :-1, i]
        ab[1, :] = b[0, :, i]
        ab[2, :-1] = a[0, 1:, i]
        ref = scipy.linalg.solve_banded((1, 1), ab, d[0, :, i])
        assert rel_inf(x[0, :, i], ref) <= 1e-10 / max(k2[i], 1.0) + 1e-12
        assert rel_inf(x[0, :, i], xl[0, :, i]) <= 1e-10 / max(k2[i], 1.0) + 1e-12


# ----------------------------------------------------------------------------------------------
# P2 manufactured solutions, P3 residual
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("shape", [(2, 64, 5), (1, 257, 3), (3, 1024, 2)])
def test_p2_manufactured_solution(shape):
    rng = np.random.default_rng(sum(shape))
    nz, ny, nx = shape
    a, b, c, _ = random_lines(rng, nz, ny, nx)
    xstar = rng.uniform(-1, 1, shape)
    d = apply_ld(a, b, c, xstar).astype(np.float64)
    for precision in ("f64", "ld"):
        x = oracle.solve_y(a, b, c, d, precision)
        err = oracle.normwise_error(x, xstar)
        assert err.max() <= 5e-15                     # cond <= ~3.5 for these lines
    # the oracle's own A x evaluator agrees with the numpy long double one
    assert np.array_equal(oracle.apply_y(a, b, c, xstar), d)


def test_p3_residual_and_evaluator():
    rng = np.random.default_rng(5)
    a, b, c, d = random_lines(rng, 2, 96, 7)
    x = oracle.solve_y(a, b, c, d)
    r_here = np.max(np.abs(apply_ld(a, b, c, x) - d.astype(LD)), axis=1).astype(np.float64)
    res, dinf, xinf, ainf = oracle.residual_y(a, b, c, d, x)
    assert np.allclose(res, r_here, rtol=1e-6, atol=1e-19)
    assert np.allclose(dinf, np.max(np.abs(d), axis=1))
    assert np.allclose(xinf, np.max(np.abs(x), axis=1))
    a0 = a.copy(); a0[:, 0, :] = 0
    c0 = c.copy(); c0[:, -1, :] = 0
    assert np.allclose(ainf, np.max(np.abs(a0) + np.abs(b) + np.abs(c0), axis=1))
    assert (res <= 1e-15 * np.maximum(dinf, 1e-300) * 10).all()      # literal bound, dominant lines
    # a deliberately wrong x is seen by the evaluator
    xb = x.copy(); xb[0, 10, 3] += 1e-6
    res_b = oracle.residual_y(a, b, c, d, xb)[0]
    assert res_b[0, 3] > 1e-7


# ----------------------------------------------------------------------------------------------
# P4 Toeplitz closed forms
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("alpha", [0.1, 1.0, 7.3])
@pytest.mark.parametrize("n", [8, 64, 512])
def test_p4_toeplitz_eigenform(alpha, n):
    """d_j = sin(pi q j/(n+1)), j=1..n  =>  x = d / lambda_q,
    lambda_q = 1 + 2 alpha - 2 alpha cos(pi q/(n+1))."""
    qs = [1, 2, n // 2, n]
    nx = len(qs)
    j = np.arange(1, n + 1, dtype=LD)
    a = np.full((1, n, nx), -alpha)
    c = np.full((1, n, nx), -alpha)
    b = np.full((1, n, nx), 1 + 2 * alpha)
    d = np.zeros((1, n, nx))
    ref = np.zeros((1, n, nx))
    for col, q in enumerate(qs):
        mode = np.sin(PI_LD * q * j / (n + 1))
        lam = 1 + 2 * LD(alpha) - 2 * LD(alpha) * np.cos(PI_LD * q / (n + 1))
        d[0, :, col] = mode.astype(np.float64)
        ref[0, :, col] = (d[0, :, col].astype(LD) / lam).astype(np.float64)
    x = oracle.solve_y(a, b, c, d)
    # d was rounded to fp64 before the solve, so compare against d/lambda of the ROUNDED d
    # up to the perturbation a 1-ulp change of d produces: cond <= 1 + 4 alpha.
    tol = (1 + 4 * alpha) * 4e-16 * 8
    assert oracle.normwise_error(x, ref).max() <= tol


@pytest.mark.parametrize("alpha", [0.1, 1.0, 9.9])
def test_p4_toeplitz_greens_function(alpha):
    """d = e_q  =>  x_j = (r^-lo - r^lo)(r^-(n+1-hi) - r^(n+1-hi)) /
                          (alpha (r^-1 - r)(r^-(n+1) - r^(n+1))),  lo/hi = min/max(j,q),
    r the root < 1 of alpha r^2 - (1+2 alpha) r + alpha = 0  (1-based j, q)."""
    n = 40
    qs = [1, 7, 20, 40]
    al = LD(alpha)
    r = ((1 + 2 * al) - np.sqrt((1 + 2 * al) ** 2 - 4 * al * al)) / (2 * al)
    nx = len(qs)
    a = np.full((1, n, nx), -alpha)
    c = np.full((1, n, nx), -alpha)
    b = np.full((1, n, nx), 1 + 2 * alpha)
    d = np.zeros((1, n, nx))
    ref = np.zeros((1, n, nx))
    for col, q in enumerate(qs):
        d[0, q - 1, col] = 1.0
        for j in range(1, n + 1):
            lo, hi = min(j, q), max(j, q)
            num = (r ** (-lo) - r ** lo) * (r ** (-(n + 1 - hi)) - r ** (n + 1 - hi))
            den = al * (1 / r - r) * (r ** (-(n + 1)) - r ** (n + 1))
            ref[0, j - 1, col] = float(num / den)
    x = oracle.solve_y(a, b, c, d)
    assert oracle.normwise_error(x, ref).max() <= 2e-14


def test_p4_second_difference_inverse_golden():
    """tests/golden/second_difference_inverse.txt: (tridiag(-1,2,-1))^-1_{ij} =
    min(i,j)(n+1-max(i,j))/(n+1), stored as exact integers over (n+1)."""
    path = os.path.join(HERE, "golden", "second_difference_inverse.txt")
    rows = [ln.split() for ln in open(path) if ln.strip() and not ln.startswith("#")]
    n = int(rows[0][0])
    numer = np.array([[int(v) for v in r] for r in rows[1:1 + n]], dtype=np.float64)
    assert numer.shape == (n, n)
    a = np.full((1, n, n), -1.0)
    c = np.full((1, n, n), -1.0)
    b = np.full((1, n, n), 2.0)
    d = np.zeros((1, n, n))
    for q in range(n):
        d[0, q, q] = 1.0                    # column q of the identity as RHS of line q
    x = oracle.solve_y(a, b, c, d)[0]       # x[:, q] = column q of the inverse
    assert np.max(np.abs(x * (n + 1) - numer)) <= 1e-12


# ----------------------------------------------------------------------------------------------
# P7 degenerate / plumbing cases
# ----------------------------------------------------------------------------------------------
def test_p7_identity_and_diagonal():
    rng = np.random.default_rng(9)
    shape = (2, 10, 3)
    d = rng.uniform(-1, 1, shape)
    z = np.zeros(shape)
    assert np.array_equal(oracle.solve_y(z, np.ones(shape), z, d), d)
    b = rng.uniform(1, 2, shape)
    assert np.array_equal(oracle.solve_y(z, b, z, d), d / b)


def test_p7_ignored_corner_entries():
    rng = np.random.default_rng(10)
    a, b, c, d = random_lines(rng, 2, 12, 3)
    x0 = oracle.solve_y(a, b, c, d)
    a2, c2 = a.copy(), c.copy()
    a2[:, 0, :] = np.nan
    c2[:, -1, :] = np.inf
    assert np.array_equal(oracle.solve_y(a2, b, c2, d), x0)
    assert np.array_equal(oracle.solve_y(a2, b, c2, d, "ld"), oracle.solve_y(a, b, c, d, "ld"))


@pytest.mark.parametrize("shape", [(1, 1, 1), (1, 2, 1), (1, 7, 1), (5, 7, 1), (1, 7, 5)])
def test_p7_small_shapes(shape):
    rng = np.random.default_rng(21)
    nz, ny, nx = shape
    a, b, c, d = random_lines(rng, nz, ny, nx)
    x = oracle.solve_y(a, b, c, d)
    for k in range(nz):
        for i in range(nx):
            A = dense_from_line(a[k, :, i], b[k, :, i], c[k, :, i]).astype(np.float64)
            assert np.allclose(A @ x[k, :, i], d[k, :, i], rtol=0, atol=1e-14)


def test_layout_is_x_fastest_lines_along_y():
    """A line-dependent matrix: the solution of line (i,k) must only see data of that line."""
    rng = np.random.default_rng(33)
    a, b, c, d = random_lines(rng, 3, 9, 4)
    x = oracle.solve_y(a, b, c, d)
    d2 = d.copy()
    d2[1, :, 2] += 1.0                                  # perturb one line only
    x2 = oracle.solve_y(a, b, c, d2)
    changed = np.any(x2 != x, axis=1)
    expect = np.zeros((3, 4), dtype=bool)
    expect[1, 2] = True
    assert np.array_equal(changed, expect)


def test_thread_count_does_not_change_bits():
    rng = np.random.default_rng(4)
    a, b, c, d = random_lines(rng, 4, 33, 9)
    nmax = oracle.max_threads()
    oracle.set_threads(1)
    x1 = oracle.solve_y(a, b, c, d)
    oracle.set_threads(nmax)
    xn = oracle.solve_y(a, b, c, d)
    assert np.array_equal(x1, xn)


# ---------------------------------------------------------------------------------------------
# f1: cyclic lines and z sweeps
# ---------------------------------------------------------------------------------------------
def _cyclic_dense(a, b, c):
    n = len(b)
    A = np.zeros((n, n))
    for j in range(n):
        A[j, j] = b[j]
        A[j, (j - 1) % n] += a[j]
        A[j, (j + 1) % n] += c[j]
    return A


@pytest.mark.parametrize("n", [3, 4, 5, 17, 32])
def test_f1_cyclic_oracle_vs_dense_lapack(n):
    rng = np.random.default_rng(100 + n)
    nx, nz = 5, 2
    a = rng.uniform(-1, 1, (nz, n, nx)); c = rng.uniform(-1, 1, (nz, n, nx))
    b = 2 + np.abs(a) + np.abs(c) + rng.uniform(0, 1, (nz, n, nx))
    d = rng.uniform(-1, 1, (nz, n, nx))
    x = oracle.solve_cyclic_y(a, b, c, d)
    for k in range(nz):
        for i in range(nx):
            ref = np.linalg.solve(_cyclic_dense(a[k, :, i], b[k, :, i], c[k, :, i]), d[k, :, i])
            assert np.max(np.abs(x[k, :, i] - ref)) <= 1e-14 * np.max(np.abs(ref))


@pytest.mark.parametrize("alpha,n", [(0.1, 16), (3.7, 64), (10.0, 512)])
def test_f1_cyclic_oracle_circulant_closed_form(alpha, n):
    """a = c = -alpha, b = 1 + 2 alpha, periodic: the matrix is circulant, its eigenvalues are
    lambda_q = 1 + 2 alpha - 2 alpha cos(2 pi q / n), so x = IFFT(FFT(d) / lambda)."""
    rng = np.random.default_rng(7)
    d = rng.uniform(-1, 1, (1, n, 3))
    a = np.full_like(d, -alpha); b = np.full_like(d, 1 + 2 * alpha)
    lam = 1 + 2 * alpha - 2 * alpha * np.cos(2 * np.pi * np.arange(n) / n)
    ref = np.fft.ifft(np.fft.fft(d, axis=1) / lam[None, :, None], axis=1).real
    x = oracle.solve_cyclic_y(a, b, a, d)
    assert np.max(np.abs(x - ref)) <= (1 + 4 * alpha) * 4e-15 * np.max(np.abs(ref))


def test_f1_solve_axis_z_is_the_transposed_problem():
    rng = np.random.default_rng(3)
    shape = (12, 5, 4)                                      # (nz, ny, nx): lines of length 12 along z
    a = rng.uniform(-1, 1, shape); c = rng.uniform(-1, 1, shape)
    b = 2 + np.abs(a) + np.abs(c); d = rng.uniform(-1, 1, shape)
    x = oracle.solve_axis(a, b, c, d, "z")
    for j in range(shape[1]):
        for i in range(shape[2]):
            ref = oracle.thomas_line(a[:, j, i], b[:, j, i], c[:, j, i], d[:, j, i])
            assert np.allclose(x[:, j, i], ref, rtol=0, atol=1e-15)
    xp = oracle.solve_axis(a, b, c, d, "z", periodic=True)
    ref = np.linalg.solve(_cyclic_dense(a[:, 2, 1], b[:, 2, 1], c[:, 2, 1]), d[:, 2, 1])
    assert np.max(np.abs(xp[:, 2, 1] - ref)) <= 1e-14


def test_f1_solve_axis_x_is_the_transposed_problem():
    rng = np.random.default_rng(4)
    shape = (3, 4, 16)                                      # lines of length 16 along x
    a = rng.uniform(-1, 1, shape); c = rng.uniform(-1, 1, shape)
    b = 2 + np.abs(a) + np.abs(c); d = rng.uniform(-1, 1, shape)
    x = oracle.solve_axis(a, b, c, d, "x")
    for k in range(shape[0]):
        for j in range(shape[1]):
            assert np.allclose(x[k, j], oracle.thomas_line(a[k, j], b[k, j], c[k, j], d[k, j]), rtol=0, atol=1e-15)
    xp = oracle.solve_axis(a, b, c, d, "x", periodic=True)
    ref = np.linalg.solve(_cyclic_dense(a[1, 2], b[1, 2], c[1, 2]), d[1, 2])
    assert np.max(np.abs(xp[1, 2] - ref)) <= 1e-14


# ----------------------------------------------------------------------------------------------
# shared coefficients, complex right-hand sides
# ----------------------------------------------------------------------------------------------
def _shared_case(rng, nz, ny, nx, cplx):
    a_y, c_y = rng.uniform(-1, 1, ny), rng.uniform(-1, 1, ny)
    b0_y = 2.5 + rng.uniform(0, 1, ny)
    sx, sz = -rng.uniform(0, 2, nx), -rng.uniform(0, 2, nz)         # b = b0 - (sx + sz) >= 2.5
    d = rng.normal(size=(nz, ny, nx))
    if cplx:
        d = d + 1j * rng.normal(size=(nz, ny, nx))
    return a_y, b0_y, c_y, sx, sz, d


def _materialise(a_y, b0_y, c_y, sx, sz, nz, ny, nx, pin00=False):
    a = np.ascontiguousarray(np.broadcast_to(a_y[None, :, None], (nz, ny, nx)))
    c = np.ascontiguousarray(np.broadcast_to(c_y[None, :, None], (nz, ny, nx)))
    b = b0_y[None, :, None] - (sx[None, None, :] + sz[:, None, None])
    if pin00:
        b[0, 0, 0] = 1.0
        c[0, 0, 0] = 0.0
    return a, b, c


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("precision", ["f64", "ld"])
@pytest.mark.parametrize("pin00", [False, True])
def test_f3_shared_equals_materialised_bit_for_bit(cplx, precision, pin00):
    rng = np.random.default_rng(31)
    nz, ny, nx = 3, 24, 5
    a_y, b0_y, c_y, sx, sz, d = _shared_case(rng, nz, ny, nx, cplx)
    x = oracle.solve_y_shared(a_y, b0_y, c_y, sx, sz, d, pin00=pin00, precision=precision)
    a, b, c = _materialise(a_y, b0_y, c_y, sx, sz, nz, ny, nx, pin00)
    assert x.dtype == d.dtype and x.shape == d.shape
    if cplx:
        assert np.array_equal(x.real, oracle.solve_y(a, b, c, d.real, precision))
        assert np.array_equal(x.imag, oracle.solve_y(a, b, c, d.imag, precision))
    else:
        assert np.array_equal(x, oracle.solve_y(a, b, c, d, precision))
    if pin00:
        assert x[0, 0, 0] == d[0, 0, 0]


@pytest.mark.parametrize("n", [2, 3, 7, 16, 32])
def test_f3_shared_complex_vs_dense_lapack(n):
    """Every line as a dense complex system (np.linalg.solve = LAPACK zgesv): a wrong shift
    index (sx/sz swapped), a shift with the wrong sign or re/im mixed up all fail here."""
    rng = np.random.default_rng(100 + n)
    nz, nx = 3, 4
    a_y, b0_y, c_y, sx, sz, d = _shared_case(rng, nz, n, nx, True)
    x = oracle.solve_y_shared(a_y, b0_y, c_y, sx, sz, d)
    for k in range(nz):
        for i in range(nx):
            A = np.zeros((n, n))
            for j in range(n):
                A[j, j] = b0_y[j] - sx[i] - sz[k]
                if j > 0:
                    A[j, j - 1] = a_y[j]
                if j < n - 1:
                    A[j, j + 1] = c_y[j]
            ref = np.linalg.solve(A.astype(np.complex128), d[k, :, i])
            assert np.max(np.abs(x[k, :, i] - ref)) <= 1e-13 * np.max(np.abs(ref))


@pytest.mark.parametrize("alpha,n", [(0.3, 17), (4.0, 64)])
def test_f3_shared_toeplitz_eigenform_with_shift(alpha, n):
    """a = c = -alpha, b0 = 1 + 2 alpha, shift s = sx + sz: d = z sin(pi q j/(n+1)) with a complex
    amplitude z is an eigenvector, x = d / (lambda_q - s)."""
    nz, nx = 2, 3
    sx, sz = -np.array([0.0, 0.5, 2.0]), -np.array([0.0, 1.25])
    j = np.arange(1, n + 1)
    d = np.empty((nz, n, nx), dtype=np.complex128)
    ref = np.empty_like(d)
    for k in range(nz):
        for i in range(nx):
            q = 1 + (3 * k + i) % n
            mode = np.sin(np.pi * q * j / (n + 1))
            lam = 1 + 2 * alpha - 2 * alpha * np.cos(np.pi * q / (n + 1))
            z = complex(1.0 + i, -2.0 + k)
            d[k, :, i] = z * mode
            ref[k, :, i] = z * mode / (lam - (sx[i] + sz[k]))
    x = oracle.solve_y_shared(np.full(n, -alpha), np.full(n, 1 + 2 * alpha), np.full(n, -alpha), sx, sz, d)
    assert np.max(np.abs(x - ref)) <= (1 + 4 * alpha) * 4e-15 * np.max(np.abs(ref))


# ----------------------------------------------------------------------------------------------
# SURVEY 8(f) f4, PDD variant
# ----------------------------------------------------------------------------------------------
def _dominant(rng, nz, ny, nx, margin=1.0):
    a, c = rng.uniform(-1, 1, (nz, ny, nx)), rng.uniform(-1, 1, (nz, ny, nx))
    b = margin + np.abs(a) + np.abs(c) + rng.uniform(0, 1, (nz, ny, nx))
    return a, b, c, rng.uniform(-1, 1, (nz, ny, nx))


@pytest.mark.parametrize("P,ny", [(2, 12), (4, 24), (3, 6)])
def test_reduced_rows_hold_for_the_exact_solution(P, ny):
    """The reduced system by definition: both rows of every partition are satisfied by the Thomas
    solution of the whole line (a wrong sign or index in the Schur complement fails here)."""
    rng = np.random.default_rng(P * 100 + ny)
    a, b, c, d = _dominant(rng, 2, ny, 3)
    x = oracle.solve_y(a, b, c, d)
    fa, fc, fd, pa, pc, pd = oracle.reduced_rows_y(a, b, c, d, P)
    m = ny // P
    for p in range(P):
        xf, xl = x[:, p * m, :], x[:, p * m + m - 1, :]
        xp = x[:, p * m - 1, :] if p > 0 else 0.0
        xn = x[:, p * m + m, :] if p < P - 1 else 0.0
        assert np.max(np.abs(fa[p] * xp + xf + fc[p] * xl - fd[p])) <= 1e-13
        assert np.max(np.abs(pa[p] * xf + xl + pc[p] * xn - pd[p])) <= 1e-13
    assert np.all(fa[0] == 0) and np.all(pc[P - 1] == 0)


def test_pdd_is_exact_when_partitions_do_not_couple_and_for_one_partition():
    rng = np.random.default_rng(7)
    a, b, c, d = _dominant(rng, 2, 32, 3)
    assert np.array_equal(oracle.solve_y_pdd(a, b, c, d, 1), oracle.solve_y(a, b, c, d))
    a2, c2 = a.copy(), c.copy()
    for p in range(1, 4):                        # cut the couplings between the 4 partitions
        a2[:, p * 8, :] = 0.0
        c2[:, p * 8 - 1, :] = 0.0
    exact = oracle.solve_y(a2, b, c2, d)
    assert np.max(np.abs(oracle.solve_y_pdd(a2, b, c2, d, 4) - exact)) <= 1e-14


def test_pdd_two_partitions_against_dense_truncation():
    """P = 2 spelled out with dense LAPACK solves: spikes from np.linalg.solve, one 2 x 2 interface
    system with the far spike ends dropped (a transposed spike or a swapped interface row fails)."""
    rng = np.random.default_rng(13)
    n, m = 12, 6
    a, b, c, d = [t[0, :, 0] for t in _dominant(rng, 1, n, 1)]
    def block(lo):
        T = np.zeros((m, m))
        for r in range(m):
            T[r, r] = b[lo + r]
            if r > 0: T[r, r - 1] = a[lo + r]
            if r < m - 1: T[r, r + 1] = c[lo + r]
        return T
    T0, T1 = block(0), block(m)
    xt0, xt1 = np.linalg.solve(T0, d[:m]), np.linalg.solve(T1, d[m:])
    e = np.zeros(m); e[m - 1] = c[m - 1]
    w0 = np.linalg.solve(T0, e)
    e = np.zeros(m); e[0] = a[m]
    v1 = np.linalg.solve(T1, e)
    yl, yf = np.linalg.solve(np.array([[1.0, w0[m - 1]], [v1[0], 1.0]]), np.array([xt0[m - 1], xt1[0]]))
    ref = np.concatenate([xt0 - w0 * yf, xt1 - v1 * yl])
    got = oracle.solve_y_pdd(a[None, :, None], b[None, :, None], c[None, :, None], d[None, :, None], 2)[0, :, 0]
    assert np.max(np.abs(got - ref)) <= 1e-14


@pytest.mark.parametrize("alpha", [0.1, 1.0, 10.0])
def test_pdd_error_decays_like_the_spikes(alpha):
    """Toeplitz ADI lines (a = c = -alpha, b = 1 + 2 alpha; BASELINE cfg 4): the dropped couplings are
    ~ r^(m-1) with r the root < 1 of alpha r^2 - (1 + 2 alpha) r + alpha = 0, so the error against the
    exact solve is bounded by a small multiple of r^(m-1) and shrinks geometrically with m."""
    rng = np.random.default_rng(11)
    r = ((1 + 2 * alpha) - np.sqrt(1 + 4 * alpha)) / (2 * alpha)
    prev = None
    for m in (4, 8, 16, 32):
        P, nz, nx = 4, 2, 3
        ny = P * m
        a = np.full((nz, ny, nx), -alpha); c = a.copy(); b = np.full((nz, ny, nx), 1 + 2 * alpha)
        d = rng.uniform(-1, 1, (nz, ny, nx))
        exact = oracle.solve_y(a, b, c, d)
        err = np.max(np.abs(oracle.solve_y_pdd(a, b, c, d, P) - exact)) / np.max(np.abs(exact))
        assert err <= 4.0 * r ** (m - 1) + 1e-15, (m, err, r ** (m - 1))
        if prev is not None and prev > 1e-13:
            assert err < prev
        prev = err
