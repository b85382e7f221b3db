// FUSED variant, TMA / pairwise-tree implementation (sm_100a).
//
// Same mapping of the paper's objects as tdma_fused.cuh (rank -> CTA of a thread-block cluster,
// MPI_Alltoall -> distributed shared memory), but built around what bounds the
// path on B200: bytes in flight and the TIME a tile occupies shared memory (resident bytes /
// tile lifetime = bandwidth).  Measured on B200 the lifetime is set by dependent-instruction
// latency (an fp64 reciprocal is a ~150-cycle chain), so the arithmetic is arranged to keep
// divisions OFF every serial chain.
//
//   * The raw a, b, c, d tile of a CTA ([R rows][TX lines] per array) is fetched by TMA tensor
//     copies (cp.async.bulk.tensor.3d) issued by one thread and completed on an mbarrier: the
//     whole tile is in flight at once, no register staging.
//   * The tile is reduced IN PLACE and the solution leaves through TMA tensor stores.
//     HBM traffic = 40 B/cell exactly (read a, b, c, d once, write x once).
//   * Leaf = M0 rows of one line, one thread.  Elimination is carried UN-NORMALISED: every row
//     is kept as  alpha x_0 + beta x_r + gamma x_{r+1} = delta  (x_0 = leaf's first unknown),
//         beta_r  = beta_{r-1} b_r - a_r gamma_{r-1},   gamma_r = beta_{r-1} c_r,
//         alpha_r = -a_r alpha_{r-1},                   delta_r = beta_{r-1} d_r - a_r delta_{r-1},
//     a chain of ONE fma per row (the textbook c'_r = c_r / (b_r - a_r c'_{r-1}) has a reciprocal
//     per row on the chain).  The per-row reciprocals 1/beta_r that back-substitution needs are
//     independent of each other and pipeline.  A second, independent sweep from the bottom
//     (eliminating the super-diagonal) produces the leaf's first-row equation
//         A x_prev + B x_0 + C x_last = D ;   the down sweep ends in  A x_0 + B x_last + C x_next = D.
//     Rows are rescaled by exact powers of two (exponent arithmetic, no rounding) so that the
//     products stay in range.  In exact arithmetic this is the modified Thomas reduction of
//     tdma_stage_kernels.cuh; only the rounding order differs.
//   * The leaf boundary equations of a line are merged PAIRWISE (binary tree, log2 W levels, one
//     thread per pair and line).  With
//         L.first: A1 x_p  + B1 x_fL + C1 x_lL = D1      R.first: A3 x_lL + B3 x_fR + C3 x_lR = D3
//         L.last : A2 x_fL + B2 x_lL + C2 x_fR = D2      R.last : A4 x_fR + B4 x_lR + C4 x_n  = D4
//     and det = B2 B3 - C2 A3, nL = B3 D2 - C2 D3, nR = B2 D3 - A3 D2, the merged node is (times det)
//         first: (det A1, det B1 - C1 B3 A2, C1 C2 C3 | det D1 - C1 nL)
//         last : (A4 A3 A2, det B4 - A4 B2 C3, det C4 | det D4 - A4 nR)
//     -- no division on the way up; the eliminated unknowns are kept as
//         x_lL = (nL - B3 A2 x_fL + C2 C3 x_lR) / det ,   x_fR = (nR + A3 A2 x_fL - B2 C3 x_lR) / det
//     whose 1/det is computed after the merged node has been handed to the next level.
//     With m0 | m = ny/P and m/m0 a power of two, the nodes of level log2(m/m0) are exactly the
//     paper's partitions and their two equations are rows 2p, 2p+1 of its reduced system (up to
//     a row scaling).
//   * The node left per (CTA, line) is ALL-GATHERED over the cluster with asynchronous DSMEM stores
//     that complete on the receiver's mbarrier (st.async ... mbarrier::complete_tx): no cluster
//     barrier on the critical path.  Every CTA solves the 2*CL-row system with the same pairwise
//     tree (a node = 2 rows) and keeps its own two boundary values; then the tree is walked
//     top-down and the leaves back-substitute from shared memory.
//
// In-place storage: a node spanning tile rows [s, e] keeps its first equation in the (A, B, C, D)
// slots of row s and its last equation in those of row e; a merge overwrites the (A, C, D) slots of
// the two eliminated unknowns with (a, c, d) of  x = d - a x_first - c x_last ; interior leaf
// rows hold (a', c', d') of  x_r = d' - a' x_0 - c' x_{r+1} ; back-substitution overwrites D with x.
#pragma once
#include <cooperative_groups.h>
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdlib.h>

namespace tdma {

namespace cg = cooperative_groups;

struct TmaFusedConfig {
    int lines = 0;      // TX
    int cluster = 0;    // CL
    int rows = 0;       // R = ny / CL
    int leaf_rows = 0;  // m0 (2, 4, 8 or 16)
    int leaves = 0;     // W = R / m0 (power of two)
    int nlev = 0;       // log2 W
    int threads = 0;    // W * TX
    int box_rows = 0;   // rows per TMA box (<= 256), divides R
    size_t smem = 0;
};

struct TmaFusedParams {
    int nx, ny, nzs;
    int CL, R, W, nlev;
    int xtiles;
    int box_rows, nbox;
#if defined(TDMA_DBG_MODE) && TDMA_DBG_MODE == 2
    long long *dbg;                     // experiment: per-CTA phase time stamps [grid][16]
#endif
};

__host__ __device__ inline size_t tma_fused_smem_bytes(int TX, int R, int CL)
{
    // tile: 4 arrays [R][TX]; cluster-level system 4 x [2 CL][TX]; two mbarriers (+ padding)
    return (size_t)4 * R * TX * sizeof(double) + (size_t)4 * 2 * CL * TX * sizeof(double) + 128;
}

namespace ptx {

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// global -> shared tile load, completes `bytes` on the mbarrier
__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *tm, int x, int y, int z, uint64_t *bar)
{
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
        ::"r"(smem_u32(dst)), "l"(tm), "r"(x), "r"(y), "r"(z), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tma_store_3d(const CUtensorMap *tm, int x, int y, int z, const void *src)
{
    asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%1, %2, %3}], [%4];"
                 ::"l"(tm), "r"(x), "r"(y), "r"(z), "r"(smem_u32(src)) : "memory");
}
__device__ __forceinline__ void tma_store_commit_and_wait_read()
{
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async_smem()
{
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
// shared::cta address -> shared::cluster address of the same offset in CTA `rank`
__device__ __forceinline__ uint32_t mapa(uint32_t addr, unsigned rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
    return r;
}
// asynchronous DSMEM store of one double that completes 8 bytes on the receiver's mbarrier
__device__ __forceinline__ void st_async_f64(uint32_t dst_cluster, double v, uint32_t bar_cluster)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.b64 [%0], %1, [%2];"
                 ::"r"(dst_cluster), "l"(__double_as_longlong(v)), "r"(bar_cluster) : "memory");
}

}  // namespace ptx

// 2^-e for |v| in [2^e, 2^(e+1)): multiplying an equation by it is exact and brings v into [1, 2)
__device__ __forceinline__ double pow2_unscale(double v)
{
    const int e = (__double2hiint(v) >> 20) & 0x7ff;
    return __hiloint2double((2046 - e) << 20, 0);
}

struct Eq { double a, b, c, d; };

__device__ __forceinline__ void eq_rescale(Eq &q)
{
    const double s = pow2_unscale(q.b);
    q.a *= s; q.b *= s; q.c *= s; q.d *= s;
}

// What a merge leaves for after the barrier: 1/det and the six numerators of the eliminated rows.
struct MergeTail { double det, p1, p2, p3, p4, nL, nR; };

// First half of a pairwise merge (see the header): rows o1 < o2 < o3 < o4 hold L.first, L.last,
// R.first, R.last; o1 / o4 receive the merged node's equations.  Division-free.
__device__ __forceinline__ MergeTail merge_head(double *__restrict__ sA, double *__restrict__ sB,
                                                double *__restrict__ sC, double *__restrict__ sD,
                                                int o1, int o2, int o3, int o4)
{
    const double A2 = sA[o2], B2 = sB[o2], C2 = sC[o2], D2 = sD[o2];
    const double A3 = sA[o3], B3 = sB[o3], C3 = sC[o3], D3 = sD[o3];
    const double A1 = sA[o1], B1 = sB[o1], C1 = sC[o1], D1 = sD[o1];
    const double A4 = sA[o4], B4 = sB[o4], C4 = sC[o4], D4 = sD[o4];
    MergeTail m;
    m.det = fma(B2, B3, -(C2 * A3));
    m.nL = fma(B3, D2, -(C2 * D3));
    m.nR = fma(B2, D3, -(A3 * D2));
    m.p1 = B3 * A2; m.p2 = C2 * C3; m.p3 = A3 * A2; m.p4 = B2 * C3;
    Eq f, l;
    f.a = m.det * A1; f.b = fma(m.det, B1, -(C1 * m.p1)); f.c = C1 * m.p2; f.d = fma(m.det, D1, -(C1 * m.nL));
    l.a = A4 * m.p3; l.b = fma(m.det, B4, -(A4 * m.p4)); l.c = m.det * C4; l.d = fma(m.det, D4, -(A4 * m.nR));
    eq_rescale(f); eq_rescale(l);
    sA[o1] = f.a; sB[o1] = f.b; sC[o1] = f.c; sD[o1] = f.d;
    sA[o4] = l.a; sB[o4] = l.b; sC[o4] = l.c; sD[o4] = l.d;
    return m;
}

// Second half: the eliminated unknowns as  x = d - a x_first - c x_last  in rows o2, o3.
__device__ __forceinline__ void merge_tail(double *__restrict__ sA, double *__restrict__ sC,
                                           double *__restrict__ sD, int o2, int o3, const MergeTail &m)
{
    const double inv = 1.0 / m.det;
    sA[o2] = m.p1 * inv; sC[o2] = -(m.p2 * inv); sD[o2] = m.nL * inv;
    sA[o3] = -(m.p3 * inv); sC[o3] = m.p4 * inv; sD[o3] = m.nR * inv;
}

__device__ __forceinline__ void unmerge_pair(const double *__restrict__ sA, const double *__restrict__ sC,
                                             double *__restrict__ sD, int o1, int o2, int o3, int o4)
{
    const double xf = sD[o1], xl = sD[o4];
    sD[o2] = fma(-sC[o2], xl, fma(-sA[o2], xf, sD[o2]));
    sD[o3] = fma(-sC[o3], xl, fma(-sA[o3], xf, sD[o3]));
}

// Pairwise tree over `nodes` nodes (a power of two) of `span` rows each, one line per lx, thread
// rows `slot` of `nslots`.  Bottom-up: on return the single remaining node has its first equation
// in row 0 and its last equation in row nodes*span-1.  Ends with a __syncthreads().
template <int TX>
__device__ __forceinline__ void tree_up(double *__restrict__ sA, double *__restrict__ sB,
                                        double *__restrict__ sC, double *__restrict__ sD,
                                        int lx, int slot, int nslots, int nodes, int span)
{
    if (nodes / 2 <= nslots) {
        // one pair per thread and level: the reciprocal of a level runs behind the next barrier
        MergeTail carry;
        int c2 = 0, c3 = 0;
        bool have = false;
        for (int n = nodes, sp = span; n > 1; n >>= 1, sp <<= 1) {
            __syncthreads();
            const bool act = slot < (n >> 1);
            MergeTail cur;
            int o2 = 0;
            if (act) {
                const int rs = slot * 2 * sp;
                o2 = (rs + sp - 1) * TX + lx;
                cur = merge_head(sA, sB, sC, sD, rs * TX + lx, o2, o2 + TX, (rs + 2 * sp - 1) * TX + lx);
            }
            if (have) merge_tail(sA, sC, sD, c2, c3, carry);
            have = act;
            if (act) { carry = cur; c2 = o2; c3 = o2 + TX; }
        }
        if (have) merge_tail(sA, sC, sD, c2, c3, carry);
    } else {
        for (int n = nodes, sp = span; n > 1; n >>= 1, sp <<= 1) {
            __syncthreads();
            for (int q = slot; q < (n >> 1); q += nslots) {
                const int rs = q * 2 * sp;
                const int o2 = (rs + sp - 1) * TX + lx;
                const MergeTail m = merge_head(sA, sB, sC, sD, rs * TX + lx, o2, o2 + TX, (rs + 2 * sp - 1) * TX + lx);
                merge_tail(sA, sC, sD, o2, o2 + TX, m);
            }
        }
    }
    __syncthreads();
}

// Top-down: needs x_first / x_last of the root in D of row 0 / row nodes*span-1 (visible to all
// threads); ends with a __syncthreads().
template <int TX>
__device__ __forceinline__ void tree_down(const double *__restrict__ sA, const double *__restrict__ sC,
                                          double *__restrict__ sD, int lx, int slot, int nslots,
                                          int nodes, int span)
{
    for (int n = 2, sp = span * (nodes >> 1); n <= nodes; n <<= 1, sp >>= 1) {
        for (int q = slot; q < (n >> 1); q += nslots) {
            const int rs = q * 2 * sp;
            const int o2 = (rs + sp - 1) * TX + lx;
            unmerge_pair(sA, sC, sD, rs * TX + lx, o2, o2 + TX, (rs + 2 * sp - 1) * TX + lx);
        }
        __syncthreads();
    }
}

// Root of a tree: first equation  B x_f + C x_l = D  (row oF, A = 0), last equation
// A x_f + B x_l = D  (row oL, C = 0)  ->  x_f, x_l into D.
__device__ __forceinline__ void solve_root(const double *__restrict__ sA, const double *__restrict__ sB,
                                           const double *__restrict__ sC, double *__restrict__ sD, int oF, int oL)
{
    const double Bf = sB[oF], Cf = sC[oF], Df = sD[oF], Al = sA[oL], Bl = sB[oL], Dl = sD[oL];
    const double inv = 1.0 / fma(Bf, Bl, -(Cf * Al));
    sD[oL] = fma(Bf, Dl, -(Al * Df)) * inv;
    sD[oF] = fma(Bl, Df, -(Cf * Dl)) * inv;
}

// Leaf reduction of M0 rows starting at tile offset o0 (row stride TX), in place.
template <int TX, int M0>
__device__ __forceinline__ void leaf_reduce(double *__restrict__ sA, double *__restrict__ sB,
                                            double *__restrict__ sC, double *__restrict__ sD,
                                            int o0, bool first_leaf, bool last_leaf)
{
    // ---- up sweep (rows M0-2 .. 0, eliminating the super-diagonal): first-row equation
    Eq u;
    {
        const int o = o0 + (M0 - 2) * TX;
        u.a = sA[o]; u.b = sB[o]; u.c = sC[o]; u.d = sD[o];
    }
#pragma unroll
    for (int r = M0 - 3; r >= 0; --r) {
        const int o = o0 + r * TX;
        const double a = sA[o], b = sB[o], c = sC[o], d = sD[o];
        Eq n;
        n.a = u.b * a;
        n.b = fma(u.b, b, -(c * u.a));
        n.c = -(c * u.c);
        n.d = fma(-c, u.d, u.b * d);
        u = n;
        if (((M0 - 3 - r) & 3) == 3 && r > 0) eq_rescale(u);
    }
    if (first_leaf) u.a = 0.0;          // global a_0 := 0
    eq_rescale(u);

    // ---- down sweep (rows 1 .. M0-1, eliminating the sub-diagonal, x_0 kept as a parameter)
    Eq p;
    {
        const int o = o0 + TX;
        p.a = sA[o]; p.b = sB[o]; p.c = sC[o]; p.d = sD[o];
    }
#pragma unroll
    for (int r = 2; r < M0; ++r) {
        const int o = o0 + r * TX;
        const double a = sA[o], b = sB[o], c = sC[o], d = sD[o];
        {   // row r-1 is interior: x_{r-1} = d' - a' x_0 - c' x_r
            const double inv = 1.0 / p.b;
            sA[o - TX] = p.a * inv; sC[o - TX] = p.c * inv; sD[o - TX] = p.d * inv;
        }
        Eq n;
        n.b = fma(p.b, b, -(a * p.c));
        n.c = p.b * c;
        n.a = -(a * p.a);
        n.d = fma(-a, p.d, p.b * d);
        p = n;
        if ((r & 3) == 1 && r < M0 - 1) eq_rescale(p);
    }
    if (last_leaf) p.c = 0.0;           // global c_{ny-1} := 0
    eq_rescale(p);
    sA[o0] = u.a; sB[o0] = u.b; sC[o0] = u.c; sD[o0] = u.d;
    const int oe = o0 + (M0 - 1) * TX;
    sA[oe] = p.a; sB[oe] = p.b; sC[oe] = p.c; sD[oe] = p.d;
}

#if defined(TDMA_DBG_MODE) && TDMA_DBG_MODE == 2
#define TDMA_STAMP(i) do { if (threadIdx.x == 0) prm.dbg[(size_t)blockIdx.x * 16 + (i)] = clock64(); } while (0)
#else
#define TDMA_STAMP(i) do { } while (0)
#endif

template <int TX, int M0, bool kCluster, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB)
fused_tma_kernel(const __grid_constant__ CUtensorMap tm_a, const __grid_constant__ CUtensorMap tm_b,
                 const __grid_constant__ CUtensorMap tm_c, const __grid_constant__ CUtensorMap tm_d,
                 const __grid_constant__ CUtensorMap tm_x, const TmaFusedParams prm)
{
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    const int R = prm.R, CL = prm.CL, W = prm.W;
    const int arr = R * TX;
    double *__restrict__ sA = reinterpret_cast<double *>(smem_raw);
    double *__restrict__ sB = sA + arr;
    double *__restrict__ sC = sB + arr;
    double *__restrict__ sD = sC + arr;
    const int NTR = 2 * CL;                                    // rows of the cluster-level system
    const int tarr = NTR * TX;
    double *__restrict__ tA = sD + arr;                        // [NTR][TX] x 4: every CTA holds a copy
    double *__restrict__ tB = tA + tarr;
    double *__restrict__ tC = tB + tarr;
    double *__restrict__ tD = tC + tarr;
    uint64_t *bar = reinterpret_cast<uint64_t *>(tD + tarr);   // [0]: TMA tile, [1]: all-gather

    const int t = threadIdx.x;
    unsigned crank = 0;
    if (kCluster) crank = cg::this_cluster().block_rank();
    const int tile = blockIdx.x / CL;
    const int xt = tile % prm.xtiles;
    const int k = tile / prm.xtiles;
    const int lx = t % TX, leaf = t / TX;
    const int x0 = xt * TX;
    const int y0 = (int)crank * R;

    TDMA_STAMP(0);
    // ---------------- TMA: the whole raw tile in flight at once ----------------
    if (t == 0) {
        ptx::mbar_init(&bar[0], 1);
        if (kCluster) ptx::mbar_init(&bar[1], 1);
        ptx::fence_mbar_init();
        ptx::mbar_expect_tx(&bar[0], (unsigned)(4 * arr * sizeof(double)));
        for (int q = 0; q < prm.nbox; ++q) {
            const int yy = y0 + q * prm.box_rows;
            const int so = q * prm.box_rows * TX;
            ptx::tma_load_3d(sB + so, &tm_b, x0, yy, k, &bar[0]);
            ptx::tma_load_3d(sA + so, &tm_a, x0, yy, k, &bar[0]);
            ptx::tma_load_3d(sC + so, &tm_c, x0, yy, k, &bar[0]);
            ptx::tma_load_3d(sD + so, &tm_d, x0, yy, k, &bar[0]);
        }
        // the all-gather below delivers 4 doubles per (node equation, line) from every CTA
        if (kCluster) ptx::mbar_expect_tx(&bar[1], (unsigned)(4 * tarr * sizeof(double)));
    }
    __syncthreads();                    // mbarriers initialised before anyone waits on them
    // split-phase cluster barrier: "every CTA of the cluster has started and initialised its
    // all-gather mbarrier" must hold before the first remote store; the matching wait sits right
    // before the exchange, where it is satisfied long ago
    if (kCluster) asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    ptx::mbar_wait(&bar[0], 0);
    TDMA_STAMP(1);

    // ---------------- leaves ----------------
    const int o0 = leaf * M0 * TX + lx;
#if defined(TDMA_DBG_MODE) && TDMA_DBG_MODE == 1
    if (prm.nx > 0) goto store_x;       // experiment: data movement only
#endif
    {
        const int grow0 = y0 + leaf * M0;
        leaf_reduce<TX, M0>(sA, sB, sC, sD, o0, grow0 == 0, grow0 + M0 == prm.ny);
    }
    TDMA_STAMP(2);

    // ---------------- pairwise tree inside the CTA, bottom-up ----------------
    tree_up<TX>(sA, sB, sC, sD, lx, leaf, W, W, M0);
    TDMA_STAMP(4);

    // ---------------- cluster level ----------------
    // the CTA's node: first equation in row 0, last equation in row R-1
    if (!kCluster) {
        if (t < TX) solve_root(sA, sB, sC, sD, lx, (R - 1) * TX + lx);
        __syncthreads();
    } else {
        // A2B as an all-gather (the paper's MPI_Alltoall, with every rank keeping a
        // copy): asynchronous DSMEM stores that complete on the RECEIVER's mbarrier -- no cluster
        // barrier on the critical path, a CTA waits only for its own inbox
        asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
        const uint32_t tA_s = ptx::smem_u32(tA), bar_s = ptx::smem_u32(&bar[1]);
        const uint32_t plane = (uint32_t)tarr * 8u;
        for (int e = t; e < 2 * TX * CL; e += (int)blockDim.x) {
            const int dest = e / (2 * TX), r = e - dest * 2 * TX;
            const int j = r / TX, l = r - j * TX;          // j: 0 = first eq, 1 = last eq
            const int o = (j ? (R - 1) * TX : 0) + l;
            const uint32_t row = (uint32_t)(((int)crank * 2 + j) * TX + l) * 8u;
            const uint32_t dst = ptx::mapa(tA_s + row, (unsigned)dest), dbar = ptx::mapa(bar_s, (unsigned)dest);
            ptx::st_async_f64(dst, sA[o], dbar);
            ptx::st_async_f64(dst + plane, sB[o], dbar);
            ptx::st_async_f64(dst + 2 * plane, sC[o], dbar);
            ptx::st_async_f64(dst + 3 * plane, sD[o], dbar);
        }
        TDMA_STAMP(5);
        ptx::mbar_wait(&bar[1], 0);
        TDMA_STAMP(6);
        // Stage B: the 2*CL-row system, solved redundantly by every CTA with the same pairwise
        // tree (a node = 2 rows), so no second exchange is needed
        tree_up<TX>(tA, tB, tC, tD, lx, leaf, W, CL, 2);
        if (t < TX) solve_root(tA, tB, tC, tD, lx, (NTR - 1) * TX + lx);
        __syncthreads();
        tree_down<TX>(tA, tC, tD, lx, leaf, W, CL, 2);
        // B2C: my node's boundary values
        for (int e = t; e < 2 * TX; e += (int)blockDim.x) {
            const int j = e / TX, l = e - j * TX;
            sD[(j ? (R - 1) * TX : 0) + l] = tD[((int)crank * 2 + j) * TX + l];
        }
        __syncthreads();
    }
    TDMA_STAMP(7);

    // ---------------- pairwise tree inside the CTA, top-down ----------------
    tree_down<TX>(sA, sC, sD, lx, leaf, W, W, M0);
    TDMA_STAMP(8);

    // ---------------- leaves: back-substitution, x overwrites d' ----------------
    {
        const double xf = sD[o0];
        double xn = sD[o0 + (M0 - 1) * TX];
#pragma unroll
        for (int r = M0 - 2; r >= 1; --r) {
            const int o = o0 + r * TX;
            xn = fma(-sC[o], xn, fma(-sA[o], xf, sD[o]));
            sD[o] = xn;
        }
    }
    TDMA_STAMP(9);
#if defined(TDMA_DBG_MODE) && TDMA_DBG_MODE == 1
store_x:
    if (kCluster) asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
#endif
    ptx::fence_proxy_async_smem();      // generic-proxy writes of D visible to the TMA engine
    __syncthreads();
    TDMA_STAMP(10);
    if (t == 0) {
        for (int q = 0; q < prm.nbox; ++q)
            ptx::tma_store_3d(&tm_x, x0, y0 + q * prm.box_rows, k, sD + q * prm.box_rows * TX);
        ptx::tma_store_commit_and_wait_read();   // smem must stay valid until the engine has read it
    }
    TDMA_STAMP(11);
#if defined(TDMA_DBG_MODE) && TDMA_DBG_MODE == 2
    if (t == 0) {
        unsigned smid; asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
        long long gt; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(gt));
        prm.dbg[(size_t)blockIdx.x * 16 + 12] = smid;
        prm.dbg[(size_t)blockIdx.x * 16 + 13] = gt;
    }
#endif
}

// ------------------------------------------------------------------------------------------
// Host side
// ------------------------------------------------------------------------------------------
inline bool is_pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }

// Eligibility: nx even (TMA global strides are multiples of 16 B), the y extent tiles as
// CL x W x m0 with W a power of two, m0 | ny/P and (ny/P)/m0 a power of two (so that one tree
// level is the paper's partition level), the tile fits shared memory.
inline bool configure_tma_fused(TmaFusedConfig *out, int nx, int ny, int P, int want_lines,
                                int want_cluster, int want_leaf, const cudaDeviceProp &prop,
                                const char **why)
{
    if (nx % 2) { *why = "TMA path needs even nx (16-byte global strides)"; return false; }
    const int m = ny / P;
    const size_t max_smem = prop.sharedMemPerBlockOptin;
    const size_t sm_smem = prop.sharedMemPerMultiprocessor;
    TmaFusedConfig best; double best_score = -1.0;
    const int tx_opts[3] = {16, 32, 8};
    const int cl_opts[5] = {1, 2, 4, 8, 16};
    for (int ti = 0; ti < 3; ++ti) {
        const int TX = tx_opts[ti];
        if (want_lines && TX != want_lines) continue;
        if (!want_lines && TX > 8 && nx < TX) continue;
        for (int ci = 0; ci < 5; ++ci) {
            const int CL = cl_opts[ci];
            if (want_cluster && CL != want_cluster) continue;
            if (CL > 8 && !want_cluster) continue;
            if (ny % CL) continue;
            const int R = ny / CL;
            if (R % m && m % R) continue;                  // partitions and CTAs must nest
            for (int m0 = 2; m0 <= m && m0 <= R && m0 <= 16; m0 *= 2) {
                if (want_leaf && m0 != want_leaf) continue;
                if (m % m0 || !is_pow2(m / m0) || R % m0 || !is_pow2(R / m0)) continue;
                TmaFusedConfig c;
                c.lines = TX; c.cluster = CL; c.rows = R; c.leaf_rows = m0; c.leaves = R / m0;
                c.threads = c.leaves * TX;
                if (c.threads > 1024) continue;
                c.nlev = 0;
                while ((1 << c.nlev) < c.leaves) ++c.nlev;
                c.box_rows = R;
                while (c.box_rows > 256) c.box_rows /= 2;
                if (R % c.box_rows) continue;
                c.smem = tma_fused_smem_bytes(TX, R, CL);
                if (c.smem > max_smem) continue;
                long ctas = (long)(sm_smem / (c.smem + 1024));
                const long by_thr = 2048 / c.threads;
                if (by_thr < ctas) ctas = by_thr;
                if (ctas < 1) continue;
                // resident cells per SM first; then >= 3 CTAs per SM (overlap of tile phases),
                // 8-row leaves, 128 B row segments, small clusters
                const double cells = (double)ctas * R * TX;
                double score = cells + (c.threads >= 32 ? 4000.0 : 0.0) + (ctas >= 3 ? 2000.0 : 0.0) + (m0 == 8 ? 1000.0 : (m0 == 16 ? 500.0 : 0.0)) +
                               (TX == 16 ? 300.0 : (TX == 32 ? 200.0 : 0.0)) - 10.0 * CL;
                if (score > best_score) { best_score = score; best = c; }
            }
        }
    }
    if (best_score < 0) {
        *why = "no (lines, cluster, leaf) tiling with power-of-two tree fits shared memory";
        return false;
    }
    *out = best;
    return true;
}

typedef CUresult (*tdma_encode_tiled_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *,
                                         const cuuint64_t *, const cuuint64_t *, const cuuint32_t *,
                                         const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                         CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

inline tdma_encode_tiled_fn get_encode_tiled()
{
    static tdma_encode_tiled_fn fn = nullptr;
    if (!fn) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<tdma_encode_tiled_fn>(p);
    }
    return fn;
}

// fp64 [nzs][ny][nx] slab, box = [1][box_rows][TX]
inline bool make_slab_tensor_map(CUtensorMap *tm, const void *base, int nx, int ny, int nzs, int TX, int box_rows)
{
    tdma_encode_tiled_fn enc = get_encode_tiled();
    if (!enc) return false;
    cuuint64_t gdim[3] = {(cuuint64_t)nx, (cuuint64_t)ny, (cuuint64_t)nzs};
    cuuint64_t gstr[2] = {(cuuint64_t)nx * sizeof(double), (cuuint64_t)nx * ny * sizeof(double)};
    cuuint32_t box[3] = {(cuuint32_t)TX, (cuuint32_t)box_rows, 1};
    cuuint32_t estr[3] = {1, 1, 1};
    const size_t inner = (size_t)TX * sizeof(double);   // one L2 request per row segment, no over-fetch
    const CUtensorMapL2promotion promo = inner >= 256 ? CU_TENSOR_MAP_L2_PROMOTION_L2_256B
                                       : inner >= 128 ? CU_TENSOR_MAP_L2_PROMOTION_L2_128B
                                                      : CU_TENSOR_MAP_L2_PROMOTION_L2_64B;
    return enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<void *>(base), gdim, gstr, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, promo,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int TX, int M0, bool kCluster, int MAXT, int MINB>
inline cudaError_t launch_tma_inst(const TmaFusedConfig &cfg, const CUtensorMap *tm, const TmaFusedParams &prm,
                                   cudaStream_t st)
{
    auto kern = fused_tma_kernel<TX, M0, kCluster, MAXT, MINB>;
    size_t smem_bytes = cfg.smem;
#if defined(TDMA_DBG_MODE) && TDMA_DBG_MODE == 2
    if (const char *pad = getenv("TDMA_PAD")) smem_bytes += (size_t)atoi(pad);   // experiment: fewer CTAs per SM
#endif
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes);
    if (e != cudaSuccess) return e;
    if (cfg.cluster > 8) {
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        if (e != cudaSuccess) return e;
    }
    cudaLaunchConfig_t lc = {};
    lc.gridDim = dim3((unsigned)((size_t)prm.xtiles * prm.nzs * cfg.cluster));
    lc.blockDim = dim3(cfg.threads);
    lc.dynamicSmemBytes = smem_bytes;
    lc.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = cfg.cluster; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    lc.attrs = attr;
    lc.numAttrs = kCluster ? 1 : 0;
    return cudaLaunchKernelEx(&lc, kern, tm[0], tm[1], tm[2], tm[3], tm[4], prm);
}

template <int TX, int M0, bool kCluster>
inline cudaError_t launch_tma_m0(const TmaFusedConfig &cfg, const CUtensorMap *tm, const TmaFusedParams &prm,
                                 cudaStream_t st)
{
    // shared memory allows about three tiles per SM: 256-thread CTAs may use up to 85 registers
    if (cfg.threads <= 256) return launch_tma_inst<TX, M0, kCluster, 256, 3>(cfg, tm, prm, st);
    return launch_tma_inst<TX, M0, kCluster, 1024, 1>(cfg, tm, prm, st);
}

template <int TX, bool kCluster>
inline cudaError_t launch_tma_tx(const TmaFusedConfig &cfg, const CUtensorMap *tm, const TmaFusedParams &prm,
                                 cudaStream_t st)
{
    switch (cfg.leaf_rows) {
    case 2: return launch_tma_m0<TX, 2, kCluster>(cfg, tm, prm, st);
    case 4: return launch_tma_m0<TX, 4, kCluster>(cfg, tm, prm, st);
    case 8: return launch_tma_m0<TX, 8, kCluster>(cfg, tm, prm, st);
    case 16: return launch_tma_m0<TX, 16, kCluster>(cfg, tm, prm, st);
    default: return cudaErrorInvalidValue;
    }
}

// a, b, c, d, x: batch base pointers (slice 0 of the launch), 16-byte aligned.
inline cudaError_t launch_tma_fused(const TmaFusedConfig &cfg, const double *a, const double *b,
                                    const double *c, const double *d, double *x, int nx, int ny,
                                    int nzs, cudaStream_t st)
{
    CUtensorMap tm[5];
    const void *ptr[5] = {a, b, c, d, x};
    for (int i = 0; i < 5; ++i)
        if (!make_slab_tensor_map(&tm[i], ptr[i], nx, ny, nzs, cfg.lines, cfg.box_rows))
            return cudaErrorInvalidValue;
    TmaFusedParams prm;
    prm.nx = nx; prm.ny = ny; prm.nzs = nzs;
    prm.CL = cfg.cluster; prm.R = cfg.rows; prm.W = cfg.leaves; prm.nlev = cfg.nlev;
    prm.xtiles = (nx + cfg.lines - 1) / cfg.lines;
    prm.box_rows = cfg.box_rows; prm.nbox = cfg.rows / cfg.box_rows;
#if defined(TDMA_DBG_MODE) && TDMA_DBG_MODE == 2
    {
        extern long long *g_tdma_dbg;
        if (!g_tdma_dbg) cudaMalloc(&g_tdma_dbg, (size_t)1 << 28);
        prm.dbg = g_tdma_dbg;
    }
#endif
    const bool cl = cfg.cluster > 1;
    switch (cfg.lines) {
    case 32: return cl ? launch_tma_tx<32, true>(cfg, tm, prm, st) : launch_tma_tx<32, false>(cfg, tm, prm, st);
    case 16: return cl ? launch_tma_tx<16, true>(cfg, tm, prm, st) : launch_tma_tx<16, false>(cfg, tm, prm, st);
    case 8: return cl ? launch_tma_tx<8, true>(cfg, tm, prm, st) : launch_tma_tx<8, false>(cfg, tm, prm, st);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace tdma
