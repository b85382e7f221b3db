"""TEST INFRASTRUCTURE: a slow numpy stand-in for the rank-local stages of the y-slab decomposition
(include/tdma.h, tdma_slab_stage_a / _b / _c), written from the header's buffer contract and from
the DEFINITION of the reduced rows as Schur complements (independent of the order
in which a kernel eliminates), with dense LAPACK solves.  It lets the multi-rank driver
(paper_2509_03933_b200/yslab.py) run on the CPU under gloo, and it gives the GPU stage test an
independent answer for the contents of the exchange buffers.  Shares no code with the CUDA path."""
import numpy as np
import torch


def reduced_rows(a, b, c, d, first_global, last_global):
    """One partition of one line (1-D arrays of m >= 2 rows) -> (fa, fc, fd, pa, pc, pd):
       fa x_prev + x_0 + fc x_{m-1} = fd   and   pa x_0 + x_{m-1} + pc x_next = pd."""
    m = len(b)
    a = a.copy(); c = c.copy()
    if first_global:
        a[0] = 0.0
    if last_global:
        c[m - 1] = 0.0
    if m == 2:
        return a[0] / b[0], c[0] / b[0], d[0] / b[0], a[1] / b[1], c[1] / b[1], d[1] / b[1]
    # interior rows 1 .. m-2:  T x_int = d_int - a_1 x_0 e_first - c_{m-2} x_{m-1} e_last
    n = m - 2
    T = np.zeros((n, n))
    for r in range(n):
        T[r, r] = b[r + 1]
        if r > 0:
            T[r, r - 1] = a[r + 1]
        if r < n - 1:
            T[r, r + 1] = c[r + 1]
    e_f = np.zeros(n); e_f[0] = 1.0
    e_l = np.zeros(n); e_l[n - 1] = 1.0
    sol = np.linalg.solve(T, np.stack([d[1:m - 1], a[1] * e_f, c[m - 2] * e_l], axis=1))
    g, u, v = sol[:, 0], sol[:, 1], sol[:, 2]          # x_int = g - u x_0 - v x_{m-1}
    # row 0:  a_0 x_prev + b_0 x_0 + c_0 x_1 = d_0,  x_1 = g_0 - u_0 x_0 - v_0 x_{m-1}
    diag = b[0] - c[0] * u[0]
    fa, fc, fd = a[0] / diag, -c[0] * v[0] / diag, (d[0] - c[0] * g[0]) / diag
    # row m-1:  a_{m-1} x_{m-2} + b_{m-1} x_{m-1} + c_{m-1} x_next = d_{m-1}
    diag = b[m - 1] - a[m - 1] * v[n - 1]
    pa, pc, pd = -a[m - 1] * u[n - 1] / diag, c[m - 1] / diag, (d[m - 1] - a[m - 1] * g[n - 1]) / diag
    return fa, fc, fd, pa, pc, pd


class NumpySlabStages:
    """Same interface as yslab.CudaSlabStages, CPU tensors, arithmetic as defined above."""

    def __init__(self, nx, ny_local, nz, P_local, batch, rank, nranks):
        self.nx, self.ny, self.nz, self.P, self.rank, self.nranks = nx, ny_local, nz, P_local, rank, nranks
        self.m = ny_local // P_local
        self.bz = nz if batch == 0 else batch
        self.nb = (nz + self.bz - 1) // self.bz
        self.device = torch.device("cpu")
        assert (nx * self.bz) % nranks == 0 and (nx * (nz % self.bz)) % nranks == 0

    def batch_lines(self, n):
        slices = min(self.bz, self.nz - n * self.bz)
        return self.nx * slices, self.nx * slices // self.nranks

    def _line(self, n, l):
        return n * self.bz + l // self.nx, l % self.nx          # (k, i) of line l of batch n

    def stage_a(self, n, a, b, c, d, send, stream=None):
        lb, ls = self.batch_lines(n)
        out = send[: self.nranks * self.P * 6 * ls].view(self.nranks, self.P, 6, ls).numpy()
        A, B, C, D = [t.numpy() for t in (a, b, c, d)]
        ptot = self.P * self.nranks
        for l in range(lb):
            k, i = self._line(n, l)
            for p in range(self.P):
                rows = slice(p * self.m, (p + 1) * self.m)
                pg = self.rank * self.P + p
                vals = reduced_rows(A[k, rows, i], B[k, rows, i], C[k, rows, i], D[k, rows, i], pg == 0, pg == ptot - 1)
                out[l // ls, p, :, l % ls] = vals

    def stage_b(self, n, recv, yout, stream=None):
        lb, ls = self.batch_lines(n)
        ptot = self.P * self.nranks
        rin = recv[: ptot * 6 * ls].view(ptot, 6, ls).numpy()
        y = yout[: 2 * ptot * ls].view(2 * ptot, ls).numpy()
        for j in range(ls):
            M = np.eye(2 * ptot)
            rhs = np.zeros(2 * ptot)
            for pg in range(ptot):
                fa, fc, fd, pa, pc, pd = rin[pg, :, j]
                if pg > 0:
                    M[2 * pg, 2 * pg - 1] = fa
                M[2 * pg, 2 * pg + 1] = fc
                M[2 * pg + 1, 2 * pg] = pa
                if pg < ptot - 1:
                    M[2 * pg + 1, 2 * pg + 2] = pc
                rhs[2 * pg], rhs[2 * pg + 1] = fd, pd
            y[:, j] = np.linalg.solve(M, rhs)

    def stage_c(self, n, yrecv, x, stream=None):
        lb, ls = self.batch_lines(n)
        yin = yrecv[: self.nranks * 2 * self.P * ls].view(self.nranks, 2 * self.P, ls).numpy()
        X = x.numpy()
        A, B, C, D = self._abcd
        m = self.m
        for l in range(lb):
            k, i = self._line(n, l)
            for p in range(self.P):
                xf, xl = yin[l // ls, 2 * p, l % ls], yin[l // ls, 2 * p + 1, l % ls]
                r0 = p * m
                X[k, r0, i], X[k, r0 + m - 1, i] = xf, xl
                if m > 2:
                    nn = m - 2
                    T = np.zeros((nn, nn))
                    rhs = D[k, r0 + 1:r0 + m - 1, i].copy()
                    for r in range(nn):
                        T[r, r] = B[k, r0 + 1 + r, i]
                        if r > 0:
                            T[r, r - 1] = A[k, r0 + 1 + r, i]
                        if r < nn - 1:
                            T[r, r + 1] = C[k, r0 + 1 + r, i]
                    rhs[0] -= A[k, r0 + 1, i] * xf
                    rhs[nn - 1] -= C[k, r0 + m - 2, i] * xl
                    X[k, r0 + 1:r0 + m - 1, i] = np.linalg.solve(T, rhs)

    # peer mode (tdma_slab_set_peers / _stage_a_peer / _stage_b_peer): the block meant for rank q goes
    # straight into rank q's receive buffer, at the place the all-to-all would have put it
    def set_peers(self, slot, recv_of_rank, yrecv_of_rank):
        if not hasattr(self, "_peers"):
            self._peers = {}
        self._peers[slot] = (list(recv_of_rank), list(yrecv_of_rank))

    def stage_a_peer(self, n, a, b, c, d, stream=None):
        lb, ls = self.batch_lines(n)
        blk = self.P * 6 * ls
        send = torch.empty(self.nranks * blk, dtype=torch.float64)
        self.stage_a(n, a, b, c, d, send)
        for q in range(self.nranks):
            self._peers[n % 3][0][q][self.rank * blk:(self.rank + 1) * blk] = send[q * blk:(q + 1) * blk]

    def stage_b_peer(self, n, recv, stream=None):
        lb, ls = self.batch_lines(n)
        blk = 2 * self.P * ls
        yout = torch.empty(self.nranks * blk, dtype=torch.float64)
        self.stage_b(n, recv, yout)
        for q in range(self.nranks):
            self._peers[n % 3][1][q][self.rank * blk:(self.rank + 1) * blk] = yout[q * blk:(q + 1) * blk]

    def bind_inputs(self, a, b, c, d):
        """stage C of the real library reads its own scratch; the stand-in re-reads the inputs."""
        self._abcd = [t.numpy() for t in (a, b, c, d)]
