// Shared-coefficient / complex-RHS lines, sm_100a.
//
// Same recursion, same cluster mapping and same tree code as tdma_fused_tma.cuh (leaf sweep ->
// K-ary merges -> DSMEM all-gather -> cluster-level system -> top-down walk -> leaf
// back-substitution), but the matrix of a line is not read from HBM: a_j, c_j and b0_j come from
// three 1-D arrays that a CTA copies into shared memory once (its R rows), and the diagonal is
// b_j = b0_j - s with the line's shift s = sx[i] + sz[k] (formed once per line in fp64, exactly
// as include/tdma.h states it).  HBM sees d once and x once: 16 B/cell real, 32 B/cell complex.
//
// What that changes on chip:
//   * only ONE array per tile travels (d), so a ring slot holds a whole tile and the ring is
//     NA >= 2 tiles deep; the sweep writes the forward-eliminated right-hand side d' back into
//     the slot IN PLACE, back-substitution overwrites it with x, and the TMA store reads x from
//     the same slot: no staging tile, and only the matrix part (a', c') of the interior rows is
//     parked in registers (4 (M0-2) instead of 6 (M0-2) registers);
//   * NC = 2: one thread owns BOTH components of a line (a 16-byte cell), so the elimination of
//     the matrix -- every reciprocal of the path -- is done once per complex line and each
//     component only adds its 3 + 2 multiply-adds per row; the tree carries two right-hand sides
//     per equation (third node-buffer plane, NodeBuf::d1).
#pragma once
#include "tdma_fused_tma.cuh"
#include "tdma_shared.h"

namespace tdma {

struct SharedParams {
    const double *a_y, *b0_y, *c_y, *sx, *sz;
    int pin00;
    int axis_z;         // 1: lines along z (rows = tensor dim 2, slices = dim 1), as in fused_tma_kernel
    int periodic;       // cyclic lines: the wrap is resolved at the root of the recursion
    int nx, ny, nzs;
    int CL, R, W, NS;
    int xtiles, ntiles;
    int box_rows, nbox;
};

template <int NC>
struct EqN { double a, b, c, d[NC]; };

// the NC right-hand-side values of one cell at shared address a
template <int NC>
__device__ __forceinline__ void ld_rhs(uint32_t a, double (&v)[NC])
{
    if (NC == 2) { const double2 t = lds2(a); v[0] = t.x; v[NC - 1] = t.y; }
    else v[0] = lds1(a);
}
template <int NC>
__device__ __forceinline__ void st_rhs(uint32_t a, const double (&v)[NC])
{
    if (NC == 2) sts2(a, v[0], v[NC - 1]);
    else sts1(a, v[0]);
}

// A node's two boundary equations, general diagonals:
//   first:  fa x_prev + fb x_f + fc x_l = fd        last:  la x_f + lb x_l + lc x_next = ld
template <int NC>
struct NodeEq { double fa, fb, fc, fd[NC], la, lb, lc, ld[NC]; };

// The two unknowns a pairwise merge eliminates (last of the left node, first of the right node) in
// terms of the merged node's first / last unknown:  x = d[j] - a[j] x_f - c[j] x_l.
template <int NC>
struct Elim { double a[2], c[2], d[2][NC]; };

// Pairwise merge in registers (the formulas of tdma_fused_tma.cuh's header with general B): the merged
// equations are carried un-normalised and rescaled by an exact power of two; one reciprocal (of the
// 2 x 2 determinant), off the chain that produces the merged node.
template <int NC>
__device__ __forceinline__ void merge_nodes(const NodeEq<NC> &L, const NodeEq<NC> &R, NodeEq<NC> &M, Elim<NC> &E)
{
    const double det = fma(L.lb, R.fb, -(L.lc * R.fa));
    const double p2 = L.lc * R.fc, p3 = R.fa * L.la;
    M.fb = fma(det, L.fb, -(L.fc * R.fb * L.la));
    M.lb = fma(det, R.lb, -(R.la * L.lb * R.fc));
    const double sf = pow2_unscale(M.fb), sl = pow2_unscale(M.lb);
    M.fa = det * L.fa * sf; M.fb *= sf; M.fc = L.fc * p2 * sf;
    M.la = R.la * p3 * sl; M.lb *= sl; M.lc = det * R.lc * sl;
    const double inv = rcp_nr(det);
    E.a[0] = R.fb * L.la * inv; E.c[0] = -(p2 * inv);
    E.a[1] = -(p3 * inv); E.c[1] = L.lb * R.fc * inv;
#pragma unroll
    for (int q = 0; q < NC; ++q) {
        const double nL = fma(R.fb, L.ld[q], -(L.lc * R.fd[q])), nR = fma(L.lb, R.fd[q], -(R.fa * L.ld[q]));
        M.fd[q] = fma(det, L.fd[q], -(L.fc * nL)) * sf;
        M.ld[q] = fma(det, R.ld[q], -(R.la * nR)) * sl;
        E.d[0][q] = nL * inv; E.d[1][q] = nR * inv;
    }
}

// What a leaf keeps in registers between its sweep and its back-substitution: the matrix part of
// the interior rows of its K sub-leaves, x_r = d'_r - ia x_first - ic x_{r+1} (d'_r lives in the
// tile slot), and the rows the in-register merges of the sub-leaves eliminated (K = 2: one merge;
// K = 4: (0,1), (2,3), then the two pairs).
template <int M0, int NC>
struct ShLeafRegs {
    static constexpr int K = M0 >= 32 ? 4 : (M0 >= 8 ? 2 : 1);
    static constexpr int H = M0 / K;
    static constexpr int HI = H - 2;
    double ia[K][HI], ic[K][HI];
    Elim<NC> e[K > 1 ? K - 1 : 1];
};

// The K swept sub-leaves as nodes with unit diagonals, merged pairwise in registers into the leaf's
// two boundary equations.
template <int M0, int NC>
__device__ __forceinline__ void leaf_finish_sh(const double (&fa)[ShLeafRegs<M0, NC>::K], const double (&fb)[ShLeafRegs<M0, NC>::K],
                                               const double (&fc)[ShLeafRegs<M0, NC>::K], const double (&fd)[ShLeafRegs<M0, NC>::K][NC],
                                               const double (&pa)[ShLeafRegs<M0, NC>::K], const double (&pc)[ShLeafRegs<M0, NC>::K],
                                               const double (&pd)[ShLeafRegs<M0, NC>::K][NC],
                                               EqN<NC> &f, EqN<NC> &l, ShLeafRegs<M0, NC> &R)
{
    constexpr int K = ShLeafRegs<M0, NC>::K;
    NodeEq<NC> nd[K];
#pragma unroll
    for (int h = 0; h < K; ++h) {
        const double inv = rcp_nr(fb[h]);
        nd[h].fa = fa[h] * inv; nd[h].fb = 1.0; nd[h].fc = fc[h] * inv;
        nd[h].la = pa[h]; nd[h].lb = 1.0; nd[h].lc = pc[h];
#pragma unroll
        for (int q = 0; q < NC; ++q) { nd[h].fd[q] = fd[h][q] * inv; nd[h].ld[q] = pd[h][q]; }
    }
    NodeEq<NC> top;
    if constexpr (K == 1) {
        top = nd[0];
    } else if constexpr (K == 2) {
        merge_nodes<NC>(nd[0], nd[K - 1], top, R.e[0]);
    } else {
        NodeEq<NC> m01, m23;
        merge_nodes<NC>(nd[0], nd[1], m01, R.e[0]);
        merge_nodes<NC>(nd[K - 2], nd[K - 1], m23, R.e[1]);
        merge_nodes<NC>(m01, m23, top, R.e[K - 2]);
    }
    f.a = top.fa; f.b = top.fb; f.c = top.fc;
    l.a = top.la; l.b = top.lb; l.c = top.lc;
#pragma unroll
    for (int q = 0; q < NC; ++q) { f.d[q] = top.fd[q]; l.d[q] = top.ld[q]; }
}

// Modified Thomas reduction of the leaf's K sub-leaves, swept interleaved (K independent
// recurrences per thread; same arithmetic as leaf_reduce in tdma_fused_tma.cuh).  cA, cB, cC: the
// leaf's rows of a_y, b0_y, c_y in shared memory; s: the line's shift; dbase: shared address of the
// leaf's first cell, rows row_bytes apart.
template <int M0, int NC>
__device__ __forceinline__ void leaf_reduce_sh(const double *__restrict__ cA, const double *__restrict__ cB,
                                               const double *__restrict__ cC, double s, uint32_t dbase,
                                               uint32_t row_bytes, bool first_leaf, bool last_leaf, bool pin,
                                               EqN<NC> &f, EqN<NC> &l, ShLeafRegs<M0, NC> &R)
{
    constexpr int K = ShLeafRegs<M0, NC>::K, H = ShLeafRegs<M0, NC>::H;
    static_assert(H >= 4, "leaves of 4, 8, 16 or 32 rows");
    double fa[K], fb[K], fc[K], fd[K][NC], pa[K], pc[K], pd[K][NC];
#pragma unroll
    for (int h = 0; h < K; ++h) {
        const int o = h * H;
        double b0 = cB[o] - s, c0 = cC[o];
        if (h == 0 && pin) { b0 = 1.0; c0 = 0.0; }             // pinned mean mode: x_0 = d_0
        double inv = rcp_nr(b0);
        double dv[NC];
        ld_rhs<NC>(dbase + (uint32_t)o * row_bytes, dv);
        fa[h] = (h == 0 && first_leaf) ? 0.0 : cA[o] * inv;    // global a_0 := 0
        fc[h] = c0 * inv; fb[h] = 1.0;
#pragma unroll
        for (int q = 0; q < NC; ++q) fd[h][q] = dv[q] * inv;
        inv = rcp_nr(cB[o + 1] - s);
        ld_rhs<NC>(dbase + (uint32_t)(o + 1) * row_bytes, dv);
        pa[h] = cA[o + 1] * inv; pc[h] = cC[o + 1] * inv;
#pragma unroll
        for (int q = 0; q < NC; ++q) pd[h][q] = dv[q] * inv;
    }
#pragma unroll
    for (int r = 2; r < H; ++r) {
#pragma unroll
        for (int h = 0; h < K; ++h) {
            const int o = h * H + r;
            const double ar = cA[o], br = cB[o] - s;
            double cr = cC[o];
            if (r == H - 1 && h == K - 1 && last_leaf) cr = 0.0;   // global c_{ny-1} := 0
            double dr[NC];
            ld_rhs<NC>(dbase + (uint32_t)o * row_bytes, dr);
            // fold row r-1 into the first-row equation, park it for back-substitution
            fb[h] = fma(-fc[h], pa[h], fb[h]);
#pragma unroll
            for (int q = 0; q < NC; ++q) fd[h][q] = fma(-fc[h], pd[h][q], fd[h][q]);
            fc[h] = -fc[h] * pc[h];
            R.ia[h][r - 2] = pa[h]; R.ic[h][r - 2] = pc[h];
            st_rhs<NC>(dbase + (uint32_t)(o - 1) * row_bytes, pd[h]);   // d' of row r-1, in place
            const double inv = rcp_nr(fma(-ar, pc[h], br));
#pragma unroll
            for (int q = 0; q < NC; ++q) pd[h][q] = fma(-ar, pd[h][q], dr[q]) * inv;
            pc[h] = cr * inv;
            pa[h] = -(ar * pa[h]) * inv;
        }
    }
    leaf_finish_sh<M0, NC>(fa, fb, fc, fd, pa, pc, pd, f, l, R);
}

// the two unknowns a merge eliminated, from the merged node's first / last unknown
template <int NC>
__device__ __forceinline__ void elim_values(const Elim<NC> &E, const double (&xf)[NC], const double (&xl)[NC],
                                            double (&lastL)[NC], double (&firstR)[NC])
{
#pragma unroll
    for (int q = 0; q < NC; ++q) {
        lastL[q] = fma(-E.c[0], xl[q], fma(-E.a[0], xf[q], E.d[0][q]));
        firstR[q] = fma(-E.c[1], xl[q], fma(-E.a[1], xf[q], E.d[1][q]));
    }
}

// Back-substitution of the leaf given its first and last unknown: d' in the slot becomes x.
template <int M0, int NC>
__device__ __forceinline__ void leaf_back_sh(const ShLeafRegs<M0, NC> &R, const double (&xf)[NC], const double (&xl)[NC],
                                             uint32_t dbase, uint32_t row_bytes)
{
    constexpr int K = ShLeafRegs<M0, NC>::K, H = ShLeafRegs<M0, NC>::H;
    double first[K][NC], xn[K][NC];                            // xn[h] starts as the sub-leaf's last unknown
#pragma unroll
    for (int q = 0; q < NC; ++q) { first[0][q] = xf[q]; xn[K - 1][q] = xl[q]; }
    if constexpr (K == 2) {
        elim_values<NC>(R.e[0], xf, xl, xn[0], first[K - 1]);
    } else if constexpr (K == 4) {
        elim_values<NC>(R.e[K - 2], xf, xl, xn[1], first[K - 2]);          // last of (0,1), first of (2,3)
        elim_values<NC>(R.e[0], xf, xn[1], xn[0], first[1]);
        elim_values<NC>(R.e[1], first[K - 2], xl, xn[K - 2], first[K - 1]);
    }
#pragma unroll
    for (int h = 0; h < K; ++h) {
        st_rhs<NC>(dbase + (uint32_t)(h * H) * row_bytes, first[h]);
        st_rhs<NC>(dbase + (uint32_t)(h * H + H - 1) * row_bytes, xn[h]);
    }
#pragma unroll
    for (int r = H - 2; r >= 1; --r) {
#pragma unroll
        for (int h = 0; h < K; ++h) {
            const uint32_t o = dbase + (uint32_t)(h * H + r) * row_bytes;
            double dp[NC];
            ld_rhs<NC>(o, dp);
#pragma unroll
            for (int q = 0; q < NC; ++q)
                xn[h][q] = fma(-R.ic[h][r - 1], xn[h][q], fma(-R.ia[h][r - 1], first[h][q], dp[q]));
            st_rhs<NC>(o, xn[h]);
        }
    }
}

// ------------------------------------------------------------------------------------------
// x sweeps (lines along the contiguous axis; real right-hand sides, 16- or 32-row leaves).  As in
// fused_tma_kernel 16 consecutive x of one line are one 128-byte row of the box
// [leaf][line][16 x], 128-byte swizzle keyed by the line (xs_addr).  The thread reads and writes
// its row in 16-byte pairs (conflict-free per quarter warp): d' of rows 2p, 2p+1 goes back as one
// store once both are known, x likewise.  Same arithmetic, in the same order, as leaf_reduce_sh /
// leaf_back_sh<16, 1>.
// ------------------------------------------------------------------------------------------
// sub-leaf h of a leaf: 8 x = pairs 4 (h & 1) .. + 3 of the 128-byte row in 16-row box h >> 1
template <int TX>
__device__ __forceinline__ uint32_t xs_sub(uint32_t box, int l, int h, int p)
{
    return xs_addr(box + (uint32_t)(h >> 1) * (uint32_t)(TX * 128), l, 4 * (h & 1) + p);
}

template <int TX, int M0>
__device__ __forceinline__ void leaf_reduce_sh_x(const double *__restrict__ cA, const double *__restrict__ cB,
                                                 const double *__restrict__ cC, double s, uint32_t box, int l,
                                                 bool first_leaf, bool last_leaf, bool pin,
                                                 EqN<1> &f, EqN<1> &le, ShLeafRegs<M0, 1> &R)
{
    constexpr int K = ShLeafRegs<M0, 1>::K, H = ShLeafRegs<M0, 1>::H;
    static_assert(H == 8 && K >= 2, "x sweeps: 16- or 32-row leaves of 8-row sub-leaves");
    double fa[K], fb[K], fc[K], fd[K][1], pa[K], pc[K], pd[K][1], hold[K];
#pragma unroll
    for (int h = 0; h < K; ++h) {
        const int o = h * H;
        double b0 = cB[o] - s, c0 = cC[o];
        if (h == 0 && pin) { b0 = 1.0; c0 = 0.0; }
        double inv = rcp_nr(b0);
        const double2 d2 = lds2(xs_sub<TX>(box, l, h, 0));
        fa[h] = (h == 0 && first_leaf) ? 0.0 : cA[o] * inv;
        fc[h] = c0 * inv; fb[h] = 1.0; fd[h][0] = d2.x * inv;
        inv = rcp_nr(cB[o + 1] - s);
        pa[h] = cA[o + 1] * inv; pc[h] = cC[o + 1] * inv; pd[h][0] = d2.y * inv;
        hold[h] = 0.0;                                   // row 0 of the sub-leaf: overwritten by x_first
    }
#pragma unroll
    for (int p = 1; p < H / 2; ++p) {
        double2 d2[K];
#pragma unroll
        for (int h = 0; h < K; ++h) d2[h] = lds2(xs_sub<TX>(box, l, h, p));
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const int r = 2 * p + e;
#pragma unroll
            for (int h = 0; h < K; ++h) {
                const int o = h * H + r;
                const double ar = cA[o], br = cB[o] - s, dr = e ? d2[h].y : d2[h].x;
                double cr = cC[o];
                if (r == H - 1 && h == K - 1 && last_leaf) cr = 0.0;
                fb[h] = fma(-fc[h], pa[h], fb[h]);
                fd[h][0] = fma(-fc[h], pd[h][0], fd[h][0]);
                fc[h] = -fc[h] * pc[h];
                R.ia[h][r - 2] = pa[h]; R.ic[h][r - 2] = pc[h];
                if (e == 0) sts2(xs_sub<TX>(box, l, h, p - 1), hold[h], pd[h][0]);   // d' of rows r-2, r-1, in place
                else hold[h] = pd[h][0];
                const double inv = rcp_nr(fma(-ar, pc[h], br));
                pd[h][0] = fma(-ar, pd[h][0], dr) * inv;
                pc[h] = cr * inv;
                pa[h] = -(ar * pa[h]) * inv;
            }
        }
    }
#pragma unroll
    for (int h = 0; h < K; ++h) sts2(xs_sub<TX>(box, l, h, 3), hold[h], 0.0);         // d' of row H-2; row H-1 becomes x_last
    leaf_finish_sh<M0, 1>(fa, fb, fc, fd, pa, pc, pd, f, le, R);
}

template <int TX, int M0>
__device__ __forceinline__ void leaf_back_sh_x(const ShLeafRegs<M0, 1> &R, const double (&xf)[1], const double (&xl)[1],
                                               uint32_t box, int l)
{
    constexpr int K = ShLeafRegs<M0, 1>::K, H = ShLeafRegs<M0, 1>::H;
    double first[K][1], xn[K][1];
    first[0][0] = xf[0]; xn[K - 1][0] = xl[0];
    if constexpr (K == 2) {
        elim_values<1>(R.e[0], xf, xl, xn[0], first[K - 1]);
    } else {
        elim_values<1>(R.e[K - 2], xf, xl, xn[1], first[K - 2]);
        elim_values<1>(R.e[0], xf, xn[1], xn[0], first[1]);
        elim_values<1>(R.e[1], first[K - 2], xl, xn[K - 2], first[K - 1]);
    }
#pragma unroll
    for (int p = H / 2 - 1; p >= 0; --p) {
#pragma unroll
        for (int h = 0; h < K; ++h) {
            const uint32_t o = xs_sub<TX>(box, l, h, p);
            const double2 dp = lds2(o);
            double hi = xn[h][0];                                   // x of row 2p+1 (p = 3: the sub-leaf's last unknown)
            if (p < H / 2 - 1) hi = fma(-R.ic[h][2 * p], xn[h][0], fma(-R.ia[h][2 * p], first[h][0], dp.y));
            double lo = first[h][0];                                // x of row 2p (p = 0: the sub-leaf's first unknown)
            if (p > 0) lo = fma(-R.ic[h][2 * p - 1], hi, fma(-R.ia[h][2 * p - 1], first[h][0], dp.x));
            sts2(o, lo, hi);
            xn[h][0] = lo;
        }
    }
}

// ------------------------------------------------------------------------------------------
// Uniform matrix (sx = sz = NULL: every line of the launch has the SAME matrix -- the ADI momentum
// sweeps, "all systems in the batch share the same matrix A").  A thread sweeps the same
// leaf rows for every tile, so everything that depends on the matrix alone is computed ONCE per
// launch: per row the multipliers of the right-hand-side recurrences go to a shared-memory table
// (read by broadcast), per leaf the multipliers of the in-register merges go to a small record,
// and the back-substitution coefficients (ia, ic), the merges' Elim::a / ::c and the matrix part
// of the leaf's two boundary equations stay in registers across tiles.  Per tile and row that
// leaves 2 multiply-adds + 1 multiply forward and 2 multiply-adds backward: no reciprocal in the
// tile loop below the tree.  The formulas and their order are those of leaf_reduce_sh / merge_nodes
// with s = 0; x agrees with the shifted kernel for zero shifts to rounding (the compiler contracts
// the two forms differently), not bit for bit.
// ------------------------------------------------------------------------------------------
struct MergeRhs { double Rfb, Llc, Llb, Rfa, det, Lfc, sf, Rla, sl, inv; };   // what merge_nodes needs for d
constexpr int kMergeRhsDoubles = 10;

template <int M0>
struct UniLeaf {
    static constexpr int K = ShLeafRegs<M0, 1>::K;
    static constexpr int kRec = K + kMergeRhsDoubles * (K - 1);   // doubles per leaf record: invfb[K], MergeRhs[K-1]
    static constexpr int kStride = M0 + 1;                       // table rows per leaf (+1: two leaves of a warp hit different banks)
};

// matrix part of merge_nodes
__device__ __forceinline__ void merge_matrix(const NodeEq<1> &L, const NodeEq<1> &R, NodeEq<1> &M, Elim<1> &E, MergeRhs &q)
{
    const double det = fma(L.lb, R.fb, -(L.lc * R.fa));
    const double p2 = L.lc * R.fc, p3 = R.fa * L.la;
    M.fb = fma(det, L.fb, -(L.fc * R.fb * L.la));
    M.lb = fma(det, R.lb, -(R.la * L.lb * R.fc));
    const double sf = pow2_unscale(M.fb), sl = pow2_unscale(M.lb);
    M.fa = det * L.fa * sf; M.fb *= sf; M.fc = L.fc * p2 * sf;
    M.la = R.la * p3 * sl; M.lb *= sl; M.lc = det * R.lc * sl;
    const double inv = rcp_nr(det);
    E.a[0] = R.fb * L.la * inv; E.c[0] = -(p2 * inv);
    E.a[1] = -(p3 * inv); E.c[1] = L.lb * R.fc * inv;
    q.Rfb = R.fb; q.Llc = L.lc; q.Llb = L.lb; q.Rfa = R.fa; q.det = det; q.Lfc = L.fc; q.sf = sf; q.Rla = R.la; q.sl = sl; q.inv = inv;
}

// right-hand-side part of merge_nodes; q: the record's 10 doubles.  kUnit: both nodes have unit
// diagonals (merges of swept sub-leaves), as the compiler also knows in merge_nodes
template <bool kUnit>
__device__ __forceinline__ void merge_rhs(const double *__restrict__ q, double Lfd, double Lld, double Rfd, double Rld,
                                          double &Mfd, double &Mld, Elim<1> &E)
{
    const double Rfb = kUnit ? 1.0 : q[0], Llb = kUnit ? 1.0 : q[2];
    const double Llc = q[1], Rfa = q[3], det = q[4], Lfc = q[5], sf = q[6], Rla = q[7], sl = q[8], inv = q[9];
    const double nL = fma(Rfb, Lld, -(Llc * Rfd)), nR = fma(Llb, Rfd, -(Rfa * Lld));
    Mfd = fma(det, Lfd, -(Lfc * nL)) * sf;
    Mld = fma(det, Rld, -(Rla * nR)) * sl;
    E.d[0][0] = nL * inv; E.d[1][0] = nR * inv;
}

// Once per launch.  tA, tB, tC: the leaf's rows (kStride apart per leaf) holding a, b0, c on entry;
// write = true (ONE thread per leaf, after every thread has read the coefficients): they become the
// table (a_r, 1 / pivot_r, running fc_r), and rec the leaf's record.  Every thread keeps R.ia, R.ic,
// Elim::a / ::c and the matrix part of f, l.
template <int M0>
__device__ __forceinline__ void leaf_matrix_uni(double *tA, double *tB, double *tC, bool first_leaf, bool last_leaf,
                                                bool write, double *rec, EqN<1> &f, EqN<1> &l, ShLeafRegs<M0, 1> &R)
{
    constexpr int K = ShLeafRegs<M0, 1>::K, H = ShLeafRegs<M0, 1>::H;
    double fa[K], fb[K], fc[K], pa[K], pc[K];
#pragma unroll
    for (int h = 0; h < K; ++h) {
        const int o = h * H;
        double inv = rcp_nr(tB[o]);
        fa[h] = (h == 0 && first_leaf) ? 0.0 : tA[o] * inv;
        fc[h] = tC[o] * inv; fb[h] = 1.0;
        if (write) tB[o] = inv;
        inv = rcp_nr(tB[o + 1]);
        pa[h] = tA[o + 1] * inv; pc[h] = tC[o + 1] * inv;
        if (write) tB[o + 1] = inv;
    }
#pragma unroll
    for (int r = 2; r < H; ++r) {
#pragma unroll
        for (int h = 0; h < K; ++h) {
            const int o = h * H + r;
            const double ar = tA[o], br = tB[o];
            double cr = tC[o];
            if (r == H - 1 && h == K - 1 && last_leaf) cr = 0.0;
            fb[h] = fma(-fc[h], pa[h], fb[h]);
            if (write) tC[o] = fc[h];                               // the fc that folds d'_{r-1} into the first equation
            fc[h] = -fc[h] * pc[h];
            R.ia[h][r - 2] = pa[h]; R.ic[h][r - 2] = pc[h];
            const double inv = rcp_nr(fma(-ar, pc[h], br));
            if (write) tB[o] = inv;
            pc[h] = cr * inv;
            pa[h] = -(ar * pa[h]) * inv;
        }
    }
    NodeEq<1> nd[K];
#pragma unroll
    for (int h = 0; h < K; ++h) {
        const double inv = rcp_nr(fb[h]);
        nd[h].fa = fa[h] * inv; nd[h].fb = 1.0; nd[h].fc = fc[h] * inv;
        nd[h].la = pa[h]; nd[h].lb = 1.0; nd[h].lc = pc[h];
        nd[h].fd[0] = 0.0; nd[h].ld[0] = 0.0;
        if (write) rec[h] = inv;
    }
    NodeEq<1> top;
    MergeRhs q[K > 1 ? K - 1 : 1];
    if constexpr (K == 1) {
        top = nd[0];
    } else if constexpr (K == 2) {
        merge_matrix(nd[0], nd[K - 1], top, R.e[0], q[0]);
    } else {
        NodeEq<1> m01, m23;
        merge_matrix(nd[0], nd[1], m01, R.e[0], q[0]);
        merge_matrix(nd[K - 2], nd[K - 1], m23, R.e[1], q[1]);
        merge_matrix(m01, m23, top, R.e[K - 2], q[K - 2]);
    }
    if (write) {
#pragma unroll
        for (int j = 0; j < K - 1; ++j) {
            double *w = rec + K + kMergeRhsDoubles * j;
            w[0] = q[j].Rfb; w[1] = q[j].Llc; w[2] = q[j].Llb; w[3] = q[j].Rfa; w[4] = q[j].det;
            w[5] = q[j].Lfc; w[6] = q[j].sf; w[7] = q[j].Rla; w[8] = q[j].sl; w[9] = q[j].inv;
        }
    }
    f.a = top.fa; f.b = top.fb; f.c = top.fc; l.a = top.la; l.b = top.lb; l.c = top.lc;
}

// the K sub-leaves' right-hand sides (fd, pd after the sweep) -> the leaf's f.d, l.d and Elim::d
template <int M0>
__device__ __forceinline__ void leaf_finish_uni(const double *__restrict__ rec, const double (&fd)[ShLeafRegs<M0, 1>::K],
                                                const double (&pd)[ShLeafRegs<M0, 1>::K], EqN<1> &f, EqN<1> &l, ShLeafRegs<M0, 1> &R)
{
    constexpr int K = ShLeafRegs<M0, 1>::K;
    double nfd[K];
#pragma unroll
    for (int h = 0; h < K; ++h) nfd[h] = fd[h] * rec[h];
    if constexpr (K == 1) {
        f.d[0] = nfd[0]; l.d[0] = pd[0];
    } else if constexpr (K == 2) {
        merge_rhs<true>(rec + K, nfd[0], pd[0], nfd[K - 1], pd[K - 1], f.d[0], l.d[0], R.e[0]);
    } else {
        double fd01, ld01, fd23, ld23;
        merge_rhs<true>(rec + K, nfd[0], pd[0], nfd[1], pd[1], fd01, ld01, R.e[0]);
        merge_rhs<true>(rec + K + kMergeRhsDoubles, nfd[K - 2], pd[K - 2], nfd[K - 1], pd[K - 1], fd23, ld23, R.e[1]);
        merge_rhs<false>(rec + K + kMergeRhsDoubles * (K - 2), fd01, ld01, fd23, ld23, f.d[0], l.d[0], R.e[K - 2]);
    }
}

// Per tile: the right-hand-side recurrences of leaf_reduce_sh with the table's multipliers.
template <int M0>
__device__ __forceinline__ void leaf_rhs_uni(const double *__restrict__ tA, const double *__restrict__ tB,
                                             const double *__restrict__ tC, const double *__restrict__ rec, uint32_t dbase,
                                             uint32_t row_bytes, EqN<1> &f, EqN<1> &l, ShLeafRegs<M0, 1> &R)
{
    constexpr int K = ShLeafRegs<M0, 1>::K, H = ShLeafRegs<M0, 1>::H;
    double fd[K], pd[K];
#pragma unroll
    for (int h = 0; h < K; ++h) {
        const int o = h * H;
        fd[h] = lds1(dbase + (uint32_t)o * row_bytes) * tB[o];
        pd[h] = lds1(dbase + (uint32_t)(o + 1) * row_bytes) * tB[o + 1];
    }
#pragma unroll
    for (int r = 2; r < H; ++r) {
#pragma unroll
        for (int h = 0; h < K; ++h) {
            const int o = h * H + r;
            const double dr = lds1(dbase + (uint32_t)o * row_bytes);
            fd[h] = fma(-tC[o], pd[h], fd[h]);
            sts1(dbase + (uint32_t)(o - 1) * row_bytes, pd[h]);     // d' of row r-1, in place
            pd[h] = fma(-tA[o], pd[h], dr) * tB[o];
        }
    }
    leaf_finish_uni<M0>(rec, fd, pd, f, l, R);
}

// the same for x sweeps (16-byte pairs through the swizzled boxes, as leaf_reduce_sh_x)
template <int TX, int M0>
__device__ __forceinline__ void leaf_rhs_uni_x(const double *__restrict__ tA, const double *__restrict__ tB,
                                               const double *__restrict__ tC, const double *__restrict__ rec, uint32_t box, int l_,
                                               EqN<1> &f, EqN<1> &l, ShLeafRegs<M0, 1> &R)
{
    constexpr int K = ShLeafRegs<M0, 1>::K, H = ShLeafRegs<M0, 1>::H;
    static_assert(H == 8 && K >= 2, "x sweeps: 16- or 32-row leaves of 8-row sub-leaves");
    double fd[K], pd[K], hold[K];
#pragma unroll
    for (int h = 0; h < K; ++h) {
        const int o = h * H;
        const double2 d2 = lds2(xs_sub<TX>(box, l_, h, 0));
        fd[h] = d2.x * tB[o]; pd[h] = d2.y * tB[o + 1];
        hold[h] = 0.0;
    }
#pragma unroll
    for (int p = 1; p < H / 2; ++p) {
        double2 d2[K];
#pragma unroll
        for (int h = 0; h < K; ++h) d2[h] = lds2(xs_sub<TX>(box, l_, h, p));
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const int r = 2 * p + e;
#pragma unroll
            for (int h = 0; h < K; ++h) {
                const int o = h * H + r;
                const double dr = e ? d2[h].y : d2[h].x;
                fd[h] = fma(-tC[o], pd[h], fd[h]);
                if (e == 0) sts2(xs_sub<TX>(box, l_, h, p - 1), hold[h], pd[h]);
                else hold[h] = pd[h];
                pd[h] = fma(-tA[o], pd[h], dr) * tB[o];
            }
        }
    }
#pragma unroll
    for (int h = 0; h < K; ++h) sts2(xs_sub<TX>(box, l_, h, 3), hold[h], 0.0);
    leaf_finish_uni<M0>(rec, fd, pd, f, l, R);
}

// Threads: leaf = t / TX, lx = t % TX; the last warp issues the TMA copies and takes no part in
// the tree (as in fused_tma_kernel).  Ring: tile q of the cluster lives in slot q % NA from its
// load until the TMA store of its x has read the slot; then tile q + NA is loaded into it.
template <int TX, int M0, bool kCluster, int MAXT, int NC, int MINB, bool kX = false, bool kUni = false>
__global__ void __launch_bounds__(MAXT, MINB)
shared_tma_kernel(const __grid_constant__ CUtensorMap tm_d, const __grid_constant__ CUtensorMap tm_x,
                  const SharedParams prm)
{
    static_assert(!kX || ((M0 == 16 || M0 == 32) && NC == 1 && TX % 8 == 0), "x sweeps: real right-hand sides, leaves of whole 128-byte rows");
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    constexpr int TXD = TX * NC;                                      // doubles per tile row
    const int R = prm.R, CL = prm.CL, W = prm.W, NA = prm.NS;
    const int arr = R * TXD;
    double *const raw = reinterpret_cast<double *>(smem_raw);         // NA slots of [R][TX][NC]
    static_assert(!kUni || (NC == 1 && M0 >= 8), "uniform matrix: real right-hand sides, leaves of 8 rows or more");
    // coefficient rows of the CTA; uniform matrix: one spare row per leaf (bank spread), then the
    // leaves' records (shared_coef_doubles on the host side is the same sum)
    constexpr int kRec = UniLeaf<M0 >= 8 ? M0 : 8>::kRec;
    const int LS = kUni ? M0 + 1 : M0, CR = kUni ? R + W : R;
    double *const cA = raw + (size_t)NA * arr, *const cB = cA + CR, *const cC = cB + CR;
    double *const rec0 = cC + CR;
    const int coef_doubles = kUni ? ((3 * CR + W * kRec + 1) & ~1) : 3 * R;
    NodeBuf nb;                                                       // node buffer: [2W][TX] per plane
    nb.ab = ptx::smem_u32(cA + coef_doubles); nb.plane = (uint32_t)(2 * W * TX) * 16u; nb.d1 = nb.ab + 2u * nb.plane;
    const uint32_t nb_bytes = 2u * nb.plane + (NC == 2 ? (uint32_t)(2 * W * TX) * 8u : 0u);
    const int NTR = 2 * CL;                                           // rows of the cluster-level system
    NodeBuf tb0;                                                      // inbox of parity 0: [NTR][TX] per plane
    tb0.ab = nb.ab + nb_bytes; tb0.plane = (uint32_t)(NTR * TX) * 16u; tb0.d1 = tb0.ab + 2u * tb0.plane;
    const uint32_t inbox_bytes = kCluster ? 2u * tb0.plane + (NC == 2 ? (uint32_t)(NTR * TX) * 8u : 0u) : 0u;
    uint64_t *bar = reinterpret_cast<uint64_t *>(smem_raw + (tb0.ab + 2u * inbox_bytes - ptx::smem_u32(smem_raw)));
    // bar[0 .. NA-1]: slot full; bar[NA], bar[NA+1]: inboxes

    const int t = threadIdx.x;
    const int NT = W * TX;
    const bool act = t < NT;
    const int tree_threads = (int)blockDim.x > 32 ? (int)blockDim.x - 32 : NT;
    const bool tree = t < tree_threads && act;
    const int Wt = tree_threads / TX;
    const unsigned tmask = __ballot_sync(0xffffffffu, tree);
    unsigned crank = 0;
    if (kCluster) crank = cg::this_cluster().block_rank();
    const int g = blockIdx.x / CL, NC_ = gridDim.x / CL;       // cluster index / number of clusters
    const int y0 = (int)crank * R;

    if (t == 0) {
        for (int i = 0; i < NA + 2; ++i) ptx::mbar_init(&bar[i], 1);
        ptx::fence_mbar_init();
    }
    for (int r = t; r < R; r += (int)blockDim.x) {             // this CTA's rows of the 1-D coefficients
        const int pr = kUni ? r + r / M0 : r;
        cA[pr] = prm.a_y[y0 + r]; cB[pr] = prm.b0_y[y0 + r]; cC[pr] = prm.c_y[y0 + r];
    }
    __syncthreads();
    if (kCluster) asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");

    const int issue_lane = t - ((int)blockDim.x - 32 > 0 ? (int)blockDim.x - 32 : 0);   // >= 0: issuing warp
    const uint32_t arr_bytes = (uint32_t)(arr * sizeof(double));
    auto issue_tile = [&](int q) {                             // load of the cluster's q-th tile
        const int tile = g + q * NC_;
        if (tile >= prm.ntiles || issue_lane != 0) return;
        const int s = q % NA;
        const int x0 = (tile % prm.xtiles) * TX, k = tile / prm.xtiles;
        double *const dst = raw + (size_t)s * arr;
        ptx::mbar_expect_tx(&bar[s], arr_bytes);
        if (kX) {                                              // one box (16 x, TX lines, W leaves, 1): [leaf][line][16 x]
            ptx::tma_load_4d(dst, &tm_d, 0, x0, y0 >> 4, k, &bar[s]);
            return;
        }
        for (int b = 0; b < prm.nbox; ++b)
        {
            const int yy = y0 + b * prm.box_rows;
            ptx::tma_load_3d(dst + b * prm.box_rows * TXD, &tm_d, x0 * NC, prm.axis_z ? k : yy, prm.axis_z ? yy : k, &bar[s]);
        }
    };
    auto store_tile = [&](int q) {                             // x of the q-th tile (TMA clips a ragged x tile)
        const int tile = g + q * NC_;
        if (issue_lane == 0) {
            const int x0 = (tile % prm.xtiles) * TX, k = tile / prm.xtiles;
            const double *const src = raw + (size_t)(q % NA) * arr;
            if (kX) ptx::tma_store_4d(&tm_x, 0, x0, y0 >> 4, k, src);
            else for (int b = 0; b < prm.nbox; ++b)
            {
                const int yy = y0 + b * prm.box_rows;
                ptx::tma_store_3d(&tm_x, x0 * NC, prm.axis_z ? k : yy, prm.axis_z ? yy : k, src + b * prm.box_rows * TXD);
            }
        }
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    };
    if (issue_lane >= 0) for (int q = 0; q < NA; ++q) issue_tile(q);

    const int lx = t % TX, leaf = t / TX;
    const bool first_leaf = !prm.periodic && y0 + leaf * M0 == 0;          // cyclic lines use a_0 and c_{n-1}
    const bool last_leaf = !prm.periodic && y0 + leaf * M0 + M0 == prm.ny;
    const uint32_t row_bytes = TXD * 8u;
    // x sweep: the leaf's box of TX 128-byte rows, addressed through xs_addr(box, lx, pair)
    const uint32_t leaf_off = kX ? (uint32_t)(leaf * M0 * TX) * 8u : (uint32_t)(leaf * M0 * TXD + lx * NC) * 8u;
    // K-ary tree levels, packed as in fused_tma_kernel
    unsigned kcode = 0, ccode = 0;
    int nl = 0;
    for (int nodes = W, cum = 0; nodes > 1; ++nl) {
        const int lkb = (nodes & 3) == 0 ? 2 : 1;
        kcode |= (unsigned)lkb << (2 * nl); ccode |= (unsigned)cum << (5 * nl);
        nodes >>= lkb; cum += lkb;
    }
    auto level_k = [&](int l) { return 1 << ((kcode >> (2 * l)) & 3u); };
    auto level_S = [&](int l) { return 2 << ((ccode >> (5 * l)) & 31u); };
    auto level_groups = [&](int l) { return W >> (((ccode >> (5 * l)) & 31u) + ((kcode >> (2 * l)) & 3u)); };
    // critical / helper warps of the tree, as in fused_tma_kernel
    const int G0 = nl > 0 ? level_groups(0) : 0;
    const int rpw = TX >= 32 ? 1 : 32 / TX;
    const int crit_rows = Wt >= 2 * G0 ? 2 * G0 : (Wt >= G0 ? G0 : Wt);
    const int cw = (crit_rows + rpw - 1) / rpw;
    const bool helper_mode = nl > 0 && (int)blockDim.x > 32 && cw * 32 < tree_threads;
    const int help0 = helper_mode ? cw * rpw : Wt;
    const int nhelp = Wt - help0;
    const int mrows = helper_mode ? crit_rows : Wt;
    const int crit_threads = helper_mode ? cw * 32 : tree_threads;
    const bool crit = tree && leaf < help0, helper = tree && !crit;

    // tile -> (x tile, slice), ring slot and its mbarrier phase, advanced without divisions
    const int step_x = NC_ % prm.xtiles, step_k = NC_ / prm.xtiles;
    int xt = g % prm.xtiles, k = g / prm.xtiles, slot = 0, sphase = 0;
    auto shift_of = [&](int xt_, int k_) {                     // the line's shift
        const int gi_ = xt_ * TX + lx < prm.nx ? xt_ * TX + lx : prm.nx - 1;   // ragged x tile: lanes past nx solve a copy
        return prm.sx[gi_] + prm.sz[k_ < prm.nzs ? k_ : prm.nzs - 1];
    };
    double s_next = (!kUni && g < prm.ntiles) ? shift_of(xt, k) : 0.0;     // uniform matrix: no shift arrays
    // uniform matrix: everything that depends on the matrix alone, once per launch
    ShLeafRegs<M0, NC> uregs;
    EqN<NC> uf, ul;
    if constexpr (kUni) {
        double *const tA = cA + leaf * LS, *const tB = cB + leaf * LS, *const tC = cC + leaf * LS;
        if (act) leaf_matrix_uni<M0>(tA, tB, tC, first_leaf, last_leaf, false, nullptr, uf, ul, uregs);
        __syncthreads();                // every thread has read the coefficients: one thread per leaf turns them into the table
        if (act && lx == 0) leaf_matrix_uni<M0>(tA, tB, tC, first_leaf, last_leaf, true, rec0 + leaf * kRec, uf, ul, uregs);
        __syncthreads();
    }
    int it = 0;
    for (int tile = g; tile < prm.ntiles; tile += NC_, ++it) {
        const int par = it & 1;
        NodeBuf tb = tb0;
        tb.ab += (uint32_t)par * inbox_bytes; tb.d1 += (uint32_t)par * inbox_bytes;
        if (kCluster && t == 0)
            ptx::mbar_expect_tx(&bar[NA + par], (unsigned)(NTR * TX * (32 + 8 * (NC - 1))));
        const double s = s_next;
        const bool pin = prm.pin00 != 0 && y0 + leaf * M0 == 0 && xt * TX + lx == 0 && k == 0;
        const uint32_t dbase = ptx::smem_u32(raw + (size_t)slot * arr) + leaf_off;
        const int cur_slot = slot, cur_phase = sphase;
        // next tile's coordinates; its shift is fetched now, a whole tile period ahead of its use
        xt += step_x; k += step_k;
        if (xt >= prm.xtiles) { xt -= prm.xtiles; ++k; }
        if (++slot == NA) { slot = 0; sphase ^= 1; }
        if (!kUni && tile + NC_ < prm.ntiles) s_next = shift_of(xt, k);
        ptx::mbar_wait(&bar[cur_slot], (unsigned)cur_phase);

        // ---------------- leaves ----------------
        ShLeafRegs<M0, NC> regs;
        if (act) {
            EqN<NC> f, l;
            if constexpr (kUni) {
                f = uf; l = ul;
                const double *const tA = cA + leaf * LS, *const tB = cB + leaf * LS, *const tC = cC + leaf * LS;
                if constexpr (kX) leaf_rhs_uni_x<TX, M0>(tA, tB, tC, rec0 + leaf * kRec, dbase, lx, f, l, uregs);
                else leaf_rhs_uni<M0>(tA, tB, tC, rec0 + leaf * kRec, dbase, row_bytes, f, l, uregs);
            } else if constexpr (kX)
                leaf_reduce_sh_x<TX, M0>(cA + leaf * M0, cB + leaf * M0, cC + leaf * M0, s, dbase, lx, first_leaf, last_leaf, pin, f, l, regs);
            else
                leaf_reduce_sh<M0, NC>(cA + leaf * M0, cB + leaf * M0, cC + leaf * M0, s, dbase, row_bytes,
                                       first_leaf, last_leaf, pin, f, l, regs);
            const uint32_t of = nb_ab<TX>(nb, 2 * leaf, lx), ol = of + TX * 16u;
            sts2(of, f.a, f.b); sts2(of + nb.plane, f.c, f.d[0]);
            sts2(ol, l.a, l.b); sts2(ol + nb.plane, l.c, l.d[0]);
            if (NC == 2) { sts1(nb_d1(nb, of), f.d[NC - 1]); sts1(nb_d1(nb, ol), l.d[NC - 1]); }
        }
        __syncthreads();                // leaf equations visible; previous tile's x complete in its slot
        if (issue_lane >= 0 && it > 0) {
            store_tile(it - 1);
            asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
            issue_tile(it - 1 + NA);    // the slot the store has just read out
        }
        if (kCluster && it == 0) asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");

        // ---------------- K-ary tree inside the CTA, bottom-up ----------------
        if (helper) {
            const int h = leaf - help0;
            int cum = 0;
            for (int l = 0; l < nl; ++l) {
                const int kk = level_k(l), S = level_S(l), groups = level_groups(l);
                int gq = (h - cum) % nhelp;
                if (gq < 0) gq += nhelp;
                double ta[6], tc[6], td[6][NC];
                if (gq < groups) {
                    if (kk == 4) kmerge_tails_regs<TX, 4, NC>(nb, lx, gq, S, ta, tc, td);
                    else kmerge_tails_regs<TX, 2, NC>(nb, lx, gq, S, ta, tc, td);
                }
                named_sync(2 + l, tree_threads);
                if (gq < groups) {
                    if (kk == 4) kmerge_tails_store<TX, 4, NC>(nb, lx, gq, S, ta, tc, td);
                    else kmerge_tails_store<TX, 2, NC>(nb, lx, gq, S, ta, tc, td);
                    for (gq += nhelp; gq < groups; gq += nhelp) {
                        if (kk == 4) kmerge_tails<TX, 4, NC>(nb, lx, gq, S, 4); else kmerge_tails<TX, 2, NC>(nb, lx, gq, S, 2);
                    }
                }
                cum += groups;
            }
        }
        if (crit) {
            for (int l = 0; l < nl; ++l) {
                const int kk = level_k(l), S = level_S(l), groups = level_groups(l);
                for (int q = leaf; q < 2 * groups; q += mrows) {
                    if (q < groups) { if (kk == 4) kmerge_fwd<TX, 4, NC>(nb, lx, q, S, 4); else kmerge_fwd<TX, 2, NC>(nb, lx, q, S, 2); }
                    else { if (kk == 4) kmerge_bwd<TX, 4, NC>(nb, lx, q - groups, S, 4); else kmerge_bwd<TX, 2, NC>(nb, lx, q - groups, S, 2); }
                }
                if (helper_mode) named_arrive(2 + l, tree_threads);
                tree_sync(crit_threads, tmask);
                if (!helper_mode) {
                    for (int q = mrows - 1 - leaf; q < groups; q += mrows) {
                        if (kk == 4) kmerge_tails<TX, 4, NC>(nb, lx, q, S, 4); else kmerge_tails<TX, 2, NC>(nb, lx, q, S, 2);
                    }
                }
            }
            // ---------------- cluster level ----------------
            if (!kCluster) {
                if (leaf == 0) solve_root<TX, NC>(nb, lx, 2 * W - 1, prm.periodic != 0);
            } else {
                // all-gather of the CTA's node (the paper's MPI_Alltoall)
                const uint32_t bar_s = ptx::smem_u32(&bar[NA + par]);
                for (int e = t; e < 4 * TX * CL; e += crit_threads) {
                    const int dest = e / (4 * TX), r = e - dest * 4 * TX;
                    const int piece = r / TX, li = r - piece * TX;  // piece: AB / CD of first, AB / CD of last
                    const int j = piece >> 1;
                    const uint32_t po = (piece & 1) ? 1u : 0u;
                    const double2 v = lds2(nb_ab<TX>(nb, j ? 2 * W - 1 : 0, li) + po * nb.plane);
                    const uint32_t dst = ptx::mapa(nb_ab<TX>(tb, (int)crank * 2 + j, li) + po * tb.plane, (unsigned)dest);
                    ptx::st_async_2f64(dst, v.x, v.y, ptx::mapa(bar_s, (unsigned)dest));
                }
                if (NC == 2) {
                    for (int e = t; e < 2 * TX * CL; e += crit_threads) {
                        const int dest = e / (2 * TX), r = e - dest * 2 * TX;
                        const int j = r / TX, li = r - j * TX;
                        const double v = lds1(nb_d1(nb, nb_ab<TX>(nb, j ? 2 * W - 1 : 0, li)));
                        const uint32_t dst = ptx::mapa(nb_d1(tb, nb_ab<TX>(tb, (int)crank * 2 + j, li)), (unsigned)dest);
                        ptx::st_async_f64(dst, v, ptx::mapa(bar_s, (unsigned)dest));
                    }
                }
                if (leaf == 0) {
                    ptx::mbar_wait(&bar[NA + par], (unsigned)((it >> 1) & 1));
                    // Stage B: every CTA computes its own two unknowns of the 2 CL-row system
                    double u0[NC], u1[NC];
                    if (!prm.periodic) {
                        cluster_solve_two_sided<TX, NC>(tb, lx, NTR, 2 * (int)crank, u0, u1);
                    } else {
                        // cyclic lines: merge the CL nodes, resolve the wrap at the root, walk back
                        kmerge_fwd<TX, 0, NC>(tb, lx, 0, 2, CL);
                        kmerge_bwd<TX, 0, NC>(tb, lx, 0, 2, CL);
                        solve_root<TX, NC>(tb, lx, NTR - 1, true);
                        kmerge_tails<TX, 0, NC>(tb, lx, 0, 2, CL);
                        double rf[NC], rl[NC];
                        nb_load_donly<NC>(tb, nb_ab<TX>(tb, 0, lx), rf);
                        nb_load_donly<NC>(tb, nb_ab<TX>(tb, NTR - 1, lx), rl);
                        kmerge_value_n<TX, NC>(tb, lx, 0, 2, CL, 2 * (int)crank, rf, rl, u0);
                        kmerge_value_n<TX, NC>(tb, lx, 0, 2, CL, 2 * (int)crank + 1, rf, rl, u1);
                    }
                    // into the CTA's own rows of its INBOX, not into the node rows: other warps of
                    // this CTA may still be reading those for their sends to the peers
                    nb_store_d<NC>(tb, nb_ab<TX>(tb, 2 * (int)crank, lx), u0);
                    nb_store_d<NC>(tb, nb_ab<TX>(tb, 2 * (int)crank + 1, lx), u1);
                }
            }
        }
        __syncthreads();

        // ---------------- top-down walk + leaf back-substitution, x written in place ----------
        if (act) {
            double xf[NC], xl[NC];
            if (kCluster) {
                nb_load_donly<NC>(tb, nb_ab<TX>(tb, 2 * (int)crank, lx), xf);
                nb_load_donly<NC>(tb, nb_ab<TX>(tb, 2 * (int)crank + 1, lx), xl);
            } else {
                nb_load_donly<NC>(nb, nb_ab<TX>(nb, 0, lx), xf);
                nb_load_donly<NC>(nb, nb_ab<TX>(nb, 2 * W - 1, lx), xl);
            }
            for (int l = nl - 1; l >= 0; --l) {
                const int kk = level_k(l), S = level_S(l);
                const int node = leaf >> ((ccode >> (5 * l)) & 31u);
                const int gq = node >> ((kcode >> (2 * l)) & 3u), j = node & (kk - 1);
                double nf[NC], nla[NC];
                kmerge_value_n<TX, NC>(nb, lx, gq, S, kk, 2 * j, xf, xl, nf);
                kmerge_value_n<TX, NC>(nb, lx, gq, S, kk, 2 * j + 1, xf, xl, nla);
#pragma unroll
                for (int q = 0; q < NC; ++q) { xf[q] = nf[q]; xl[q] = nla[q]; }
            }
            if constexpr (kX) leaf_back_sh_x<TX, M0>(kUni ? uregs : regs, xf, xl, dbase, lx);
            else leaf_back_sh<M0, NC>(kUni ? uregs : regs, xf, xl, dbase, row_bytes);
            ptx::fence_proxy_async_smem();      // x in the slot -> visible to the TMA store
        }
    }
    if (it > 0) {
        __syncthreads();
        if (issue_lane >= 0) {
            store_tile(it - 1);
            asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
        }
    }
}

// ------------------------------------------------------------------------------------------
// Host side
// ------------------------------------------------------------------------------------------
inline size_t shared_smem_bytes(int TX, int R, int W, int CL, int NA, int NC, int uni_leaf = 0)
{
    const size_t slots = (size_t)NA * R * TX * NC * sizeof(double);
    // uniform matrix (uni_leaf = its leaf size): padded table rows + the leaves' records, as in the kernel
    const int rec = uni_leaf >= 32 ? UniLeaf<32>::kRec : UniLeaf<16>::kRec;
    const size_t coef = (uni_leaf ? (size_t)((3 * (R + W) + W * rec + 1) & ~1) : (size_t)3 * R) * sizeof(double);
    const size_t node = (size_t)2 * W * TX * (32 + 8 * (NC - 1));
    const size_t inbox = CL > 1 ? (size_t)2 * 2 * CL * TX * (32 + 8 * (NC - 1)) : 0;
    return slots + coef + node + inbox + 128;
}

// Leaf sizes the kernel is instantiated for.
// 24 / 12 and 20 / 10 rows (two sub-leaves of 12, 6, 10, 5) tile 3 * 2^k and 5 * 2^k line lengths (96, 192, 384, 768,
// 160, 320, 640 ...) with the same power-of-two tree; built for the default tile width only.
constexpr int kSharedLeafSizes[] = {32, 24, 20, 16, 12, 10, 8, 4};
inline bool shared_odd_leaf(int m0) { return m0 == 24 || m0 == 20 || m0 == 12 || m0 == 10; }

inline bool configure_shared_impl(SharedConfig *out, int nx, int ny, int NC, int want_lines, int want_cluster,
                                  int want_leaf, int want_slots, int want_ctas, const cudaDeviceProp &prop, const char **why,
                                  bool xsweep = false, bool uniform = false)
{
    if (uniform && NC != 1) { *why = "uniform matrix: real right-hand sides"; return false; }
    if (NC != 1 && NC != 2) { *why = "ncomp must be 1 (real) or 2 (complex)"; return false; }
    if (xsweep && (NC != 1 || ny % 16)) { *why = "x sweeps: real right-hand sides, line length a multiple of 16"; return false; }
    if (!xsweep && (nx * NC) % 2) { *why = "TMA path needs an even number of doubles per row (16-byte global strides)"; return false; }
    const size_t max_smem = prop.sharedMemPerBlockOptin;
    SharedConfig best; double best_score = -1.0;
    // lines per tile: 128-byte row segments first (16 real / 8 complex cells), then 256-byte ones
    const int tx_opts[3] = {NC == 1 ? 16 : 8, NC == 1 ? 32 : 16, NC == 1 ? 8 : 4};
    const int cl_opts[7] = {1, 2, 4, 8, 3, 6, 5};                    // 3, 6, 5: x sweeps of 3 * 2^k / 5 * 2^k cells
    for (int ti = 0; ti < 3; ++ti) {
        const int TX = tx_opts[ti];
        if (want_lines ? TX != want_lines : ti == 2) continue;      // 64-byte segments only on request
        if ((xsweep || uniform) && TX != 16) continue;              // x sweeps: 16 lines of 128-byte leaf rows
        for (int ci = 0; ci < 7; ++ci) {
            const int CL = cl_opts[ci];
            if (want_cluster && CL != want_cluster) continue;
            if ((CL == 3 || CL == 6 || CL == 5) && !xsweep) continue;
            if (ny % CL) continue;
            const int R = ny / CL;
            for (int m0 : kSharedLeafSizes) {
                if (want_leaf && m0 != want_leaf) continue;
                if ((xsweep || uniform) && m0 != 16 && m0 != 32) continue;
                if (m0 > R || R % m0 || !is_pow2(R / m0) || R / m0 > 32) continue;
                if (shared_odd_leaf(m0) && (ti != 0 || want_ctas >= 2 || (m0 >= 20 && NC != 1))) continue;
                // 32-row leaves (four sub-leaves per thread) halve the tree per cell: 1.46 -> 1.05 ms on 256 slices
                // of cfg 3 (real).  Complex cells need the registers for the second right-hand side: on request only
                if (m0 == 32 && want_leaf != 32 && NC != 1) continue;
                SharedConfig c;
                c.ncomp = NC; c.lines = TX; c.cluster = CL; c.rows = R; c.leaf_rows = m0; c.leaves = R / m0;
                c.threads = c.leaves * TX; c.xsweep = xsweep ? 1 : 0; c.uniform = uniform ? 1 : 0;
                if (uniform && c.threads > 256) continue;
                if (c.threads > 512 || ((m0 == 32 || shared_odd_leaf(m0)) && c.threads > 256)) continue;
                c.box_rows = R;
                while (c.box_rows > 256) c.box_rows /= 2;
                if (R % c.box_rows) continue;
                c.slots = 0;
                for (int na = want_slots ? want_slots : 4; na >= (want_slots ? want_slots : 2); --na) {
                    c.smem = shared_smem_bytes(TX, R, c.leaves, CL, na, NC, uniform ? m0 : 0);
                    if (c.smem <= max_smem) { c.slots = na; break; }
                }
                if (!c.slots) continue;
                c.ctas_per_sm = 1;
                if (want_ctas >= 2 && !xsweep && !uniform) {          // co-residency: registers and shared memory shared out
                    if (c.threads * want_ctas > 512 || m0 != 16) continue;
                    for (; c.slots >= 2; --c.slots) {
                        c.smem = shared_smem_bytes(TX, R, c.leaves, CL, c.slots, NC);
                        if ((size_t)want_ctas * (c.smem + 1024) <= prop.sharedMemPerMultiprocessor) break;
                    }
                    if (c.slots < 2) continue;
                    c.ctas_per_sm = want_ctas;
                }
                // as for the general kernel: long leaves (fewer tree levels) first, then 256 threads
                // per CTA (255 registers each), 128-byte segments, a deep ring, small clusters
                const double score = 10000.0 * m0 + (c.threads == 256 ? 4000.0 : (c.threads > 256 ? 1000.0 : 2000.0 + c.threads)) +
                                     (ti == 0 ? 500.0 : 0.0) + 100.0 * c.slots - 50.0 * CL;
                if (score > best_score) { best_score = score; best = c; }
            }
        }
    }
    if (best_score < 0) {
        *why = "no (lines, cluster, leaf) tiling with a power-of-two tree of <= 32 leaves of 4, 8 or 16 rows fits";
        return false;
    }
    *out = best;
    return true;
}

// d / x as a tensor of doubles (nx * NC, ny, nz), box (TX * NC, box_rows, 1)
inline bool make_shared_tensor_map(CUtensorMap *tm, const void *base, int nx, int ny, int nz, int NC, int TX, int box_rows,
                                   long long rs, long long os, bool axis_z)
{
    tdma_encode_tiled_fn enc = get_encode_tiled();
    if (!enc) return false;
    // rs / os: cells between rows of a line / between slices (y sweep: nx, nx * ny; z sweep: nx * slices, nx)
    cuuint64_t gdim[3] = {(cuuint64_t)nx * NC, (cuuint64_t)(axis_z ? nz : ny), (cuuint64_t)(axis_z ? ny : nz)};
    cuuint64_t gstr[2] = {(cuuint64_t)(axis_z ? os : rs) * NC * sizeof(double), (cuuint64_t)(axis_z ? rs : os) * NC * sizeof(double)};
    cuuint32_t box[3] = {(cuuint32_t)(TX * NC), (cuuint32_t)(axis_z ? 1 : box_rows), (cuuint32_t)(axis_z ? box_rows : 1)};
    cuuint32_t estr[3] = {1, 1, 1};
    const size_t inner = (size_t)TX * NC * sizeof(double);
    const CUtensorMapL2promotion promo = inner >= 256 ? CU_TENSOR_MAP_L2_PROMOTION_L2_256B : CU_TENSOR_MAP_L2_PROMOTION_L2_128B;
    return enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<void *>(base), gdim, gstr, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, promo,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int TX, int M0, bool kCluster, int MAXT, int NC, int MINB = 1, bool kX = false, bool kUni = false>
inline cudaError_t launch_shared_inst(SharedConfig &cfg, const CUtensorMap *tm, const SharedParams &prm, cudaStream_t st)
{
    auto kern = shared_tma_kernel<TX, M0, kCluster, MAXT, NC, MINB, kX, kUni>;
    cudaLaunchConfig_t lc = {};
    lc.blockDim = dim3((cfg.threads + 31) & ~31);
    lc.dynamicSmemBytes = cfg.smem;
    lc.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = cfg.cluster; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    lc.attrs = attr;
    lc.numAttrs = kCluster ? 1 : 0;
    if (cfg.max_clusters <= 0) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cfg.smem);
        if (e != cudaSuccess) return e;
        int dev = 0, sms = 0, n = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (kCluster) {
            lc.gridDim = dim3((unsigned)(cfg.cluster * sms));
            e = cudaOccupancyMaxActiveClusters(&n, kern, &lc);
            if (e != cudaSuccess) return e;
        } else {
            e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kern, (int)lc.blockDim.x, cfg.smem);
            if (e != cudaSuccess) return e;
            n *= sms;
        }
        if (n < 1) return cudaErrorLaunchOutOfResources;
        cfg.max_clusters = n;
    }
    if (prm.ntiles <= 0) return cudaSuccess;
    const int nc = prm.ntiles < cfg.max_clusters ? prm.ntiles : cfg.max_clusters;
    lc.gridDim = dim3((unsigned)(nc * cfg.cluster));
    return cudaLaunchKernelEx(&lc, kern, tm[0], tm[1], prm);
}

template <int TX, int NC, bool kCluster>
inline cudaError_t launch_shared_tx(SharedConfig &cfg, const CUtensorMap *tm, const SharedParams &prm, cudaStream_t st)
{
    const bool big = cfg.threads > 256;
    // co-resident CTAs: one sweeps while another walks its tree.  128-thread CTAs keep up to 255
    // (two per SM) or 168 (three) registers per thread, 256-thread CTAs 128
    if (cfg.ctas_per_sm >= 2 && cfg.leaf_rows == 16 && !big) {
        if (cfg.threads <= 128) {
            if (cfg.ctas_per_sm == 2) return launch_shared_inst<TX, 16, kCluster, 128, NC, 2>(cfg, tm, prm, st);
            if (cfg.ctas_per_sm == 3) return launch_shared_inst<TX, 16, kCluster, 128, NC, 3>(cfg, tm, prm, st);
            return launch_shared_inst<TX, 16, kCluster, 128, NC, 4>(cfg, tm, prm, st);
        }
        return launch_shared_inst<TX, 16, kCluster, 256, NC, 2>(cfg, tm, prm, st);
    }
    if constexpr ((NC == 1 && TX == 16) || (NC == 2 && TX == 8)) {        // 3 * 2^k and 5 * 2^k line lengths
        if (!big && cfg.leaf_rows == 12) return launch_shared_inst<TX, 12, kCluster, 256, NC>(cfg, tm, prm, st);
        if (!big && cfg.leaf_rows == 10) return launch_shared_inst<TX, 10, kCluster, 256, NC>(cfg, tm, prm, st);
        if constexpr (NC == 1) {
            if (!big && cfg.leaf_rows == 24) return launch_shared_inst<TX, 24, kCluster, 256, NC>(cfg, tm, prm, st);
            if (!big && cfg.leaf_rows == 20) return launch_shared_inst<TX, 20, kCluster, 256, NC>(cfg, tm, prm, st);
        }
    }
    switch (cfg.leaf_rows) {
    case 32: return big ? cudaErrorInvalidValue : launch_shared_inst<TX, 32, kCluster, 256, NC>(cfg, tm, prm, st);
    case 16: return big ? launch_shared_inst<TX, 16, kCluster, 512, NC>(cfg, tm, prm, st)
                        : launch_shared_inst<TX, 16, kCluster, 256, NC>(cfg, tm, prm, st);
    case 8: return big ? launch_shared_inst<TX, 8, kCluster, 512, NC>(cfg, tm, prm, st)
                       : launch_shared_inst<TX, 8, kCluster, 256, NC>(cfg, tm, prm, st);
    case 4: return big ? cudaErrorInvalidValue : launch_shared_inst<TX, 4, kCluster, 256, NC>(cfg, tm, prm, st);
    default: return cudaErrorInvalidValue;
    }
}

inline cudaError_t launch_shared_impl(SharedConfig &cfg, const SharedArgs &a, cudaStream_t st)
{
    CUtensorMap tm[2];
    if (a.nzs > 0 && cfg.xsweep) {
        if (!make_xsweep_tensor_map(&tm[0], a.d, a.ny, a.nx, a.nzs, cfg.lines, cfg.rows / 16) ||
            !make_xsweep_tensor_map(&tm[1], a.x, a.ny, a.nx, a.nzs, cfg.lines, cfg.rows / 16))
            return cudaErrorInvalidValue;
    } else if (a.nzs > 0) {
        if (!make_shared_tensor_map(&tm[0], a.d, a.nx, a.ny, a.nzs, cfg.ncomp, cfg.lines, cfg.box_rows, a.rs, a.os, a.axis_z != 0) ||
            !make_shared_tensor_map(&tm[1], a.x, a.nx, a.ny, a.nzs, cfg.ncomp, cfg.lines, cfg.box_rows, a.rs, a.os, a.axis_z != 0))
            return cudaErrorInvalidValue;
    }
    SharedParams prm;
    prm.a_y = a.a_y; prm.b0_y = a.b0_y; prm.c_y = a.c_y; prm.sx = a.sx; prm.sz = a.sz;
    prm.pin00 = a.pin00;
    prm.axis_z = a.axis_z; prm.periodic = a.periodic;
    prm.nx = a.nx; prm.ny = a.ny; prm.nzs = a.nzs;
    prm.CL = cfg.cluster; prm.R = cfg.rows; prm.W = cfg.leaves; prm.NS = cfg.slots;
    prm.xtiles = (a.nx + cfg.lines - 1) / cfg.lines;
    prm.ntiles = prm.xtiles * a.nzs;
    prm.box_rows = cfg.box_rows; prm.nbox = cfg.rows / cfg.box_rows;
    const bool cl = cfg.cluster > 1;
    if (cfg.uniform) {
        if (cfg.ncomp != 1 || cfg.lines != 16 || cfg.threads > 256 || !a.uniform) return cudaErrorInvalidValue;
        const bool xs = cfg.xsweep != 0;
        if (cfg.leaf_rows == 32) {
            if (xs) return cl ? launch_shared_inst<16, 32, true, 256, 1, 1, true, true>(cfg, tm, prm, st) : launch_shared_inst<16, 32, false, 256, 1, 1, true, true>(cfg, tm, prm, st);
            return cl ? launch_shared_inst<16, 32, true, 256, 1, 1, false, true>(cfg, tm, prm, st) : launch_shared_inst<16, 32, false, 256, 1, 1, false, true>(cfg, tm, prm, st);
        }
        if (cfg.leaf_rows == 16) {
            if (xs) return cl ? launch_shared_inst<16, 16, true, 256, 1, 1, true, true>(cfg, tm, prm, st) : launch_shared_inst<16, 16, false, 256, 1, 1, true, true>(cfg, tm, prm, st);
            return cl ? launch_shared_inst<16, 16, true, 256, 1, 1, false, true>(cfg, tm, prm, st) : launch_shared_inst<16, 16, false, 256, 1, 1, false, true>(cfg, tm, prm, st);
        }
        return cudaErrorInvalidValue;
    }
    if (a.uniform) return cudaErrorInvalidValue;           // NULL shift arrays need the uniform-matrix tiling
    if (cfg.xsweep) {
        if (cfg.ncomp != 1 || cfg.lines != 16 || (cfg.leaf_rows != 16 && cfg.leaf_rows != 32)) return cudaErrorInvalidValue;
        if (cfg.leaf_rows == 32)
            return cl ? launch_shared_inst<16, 32, true, 256, 1, 1, true>(cfg, tm, prm, st) : launch_shared_inst<16, 32, false, 256, 1, 1, true>(cfg, tm, prm, st);
        if (cfg.threads > 256)
            return cl ? launch_shared_inst<16, 16, true, 512, 1, 1, true>(cfg, tm, prm, st) : launch_shared_inst<16, 16, false, 512, 1, 1, true>(cfg, tm, prm, st);
        return cl ? launch_shared_inst<16, 16, true, 256, 1, 1, true>(cfg, tm, prm, st) : launch_shared_inst<16, 16, false, 256, 1, 1, true>(cfg, tm, prm, st);
    }
    if (cfg.ncomp == 1) {
        if (cfg.lines == 8) return cl ? launch_shared_tx<8, 1, true>(cfg, tm, prm, st) : launch_shared_tx<8, 1, false>(cfg, tm, prm, st);
        if (cfg.lines == 16) return cl ? launch_shared_tx<16, 1, true>(cfg, tm, prm, st) : launch_shared_tx<16, 1, false>(cfg, tm, prm, st);
        if (cfg.lines == 32) return cl ? launch_shared_tx<32, 1, true>(cfg, tm, prm, st) : launch_shared_tx<32, 1, false>(cfg, tm, prm, st);
    } else {
        if (cfg.lines == 8) return cl ? launch_shared_tx<8, 2, true>(cfg, tm, prm, st) : launch_shared_tx<8, 2, false>(cfg, tm, prm, st);
        if (cfg.lines == 16) return cl ? launch_shared_tx<16, 2, true>(cfg, tm, prm, st) : launch_shared_tx<16, 2, false>(cfg, tm, prm, st);
    }
    return cudaErrorInvalidValue;
}

}  // namespace tdma
