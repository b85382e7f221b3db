// FUSED variant, persistent TMA / pairwise-tree implementation (sm_100a).
//
// Same mapping of the paper's objects as tdma_fused.cuh (rank -> CTA of a thread-block cluster,
// MPI_Alltoall -> distributed shared memory), but built around what bounds the
// path on B200: bandwidth = bytes in flight / latency, and the bytes in flight live in shared
// memory.  So shared memory holds (almost) nothing but RAW tiles that are in flight or being
// swept, everything that has to survive the reduced-system phase is parked elsewhere:
//
//   * Persistent clusters.  A cluster of CL CTAs owns TX consecutive lines (CTA c the rows
//     c*R .. c*R+R-1, R = ny/CL) and loops over tiles (tile = x-tile, z-slice) with a static
//     stride.  The raw a, b, c, d tile of a CTA ([R][TX] per array) is fetched by TMA tensor copies
//     (cp.async.bulk.tensor.3d) completed on an mbarrier.  As soon as the leaf sweep of tile i has
//     consumed the raw buffer, the copies of tile i+1 are issued into it, so HBM latency runs
//     behind the tree / cluster phases of tile i instead of in front of them.
//   * Leaf = M0 rows of one line, one thread: modified Thomas reduction (tdma_stage_kernels.cuh)
//     from shared memory.  The forward-eliminated interior rows (a', c', d') stay in the thread's
//     REGISTERS until back-substitution; only the two boundary equations of the leaf go to a small
//     node buffer in shared memory.  x is streamed to HBM straight from registers (128-byte
//     segments per half warp).  HBM traffic = 40 B/cell exactly.
//   * The leaf boundary equations of a line are merged PAIRWISE (binary tree, log2 W levels, one
//     thread per pair and line), carried un-normalised (general diagonal B) so that no division
//     sits on the way up.  With
//         L.first: A1 x_p  + B1 x_fL + C1 x_lL = D1      R.first: A3 x_lL + B3 x_fR + C3 x_lR = D3
//         L.last : A2 x_fL + B2 x_lL + C2 x_fR = D2      R.last : A4 x_fR + B4 x_lR + C4 x_n  = D4
//     and det = B2 B3 - C2 A3, nL = B3 D2 - C2 D3, nR = B2 D3 - A3 D2, the merged node is (times det)
//         first: (det A1, det B1 - C1 B3 A2, C1 C2 C3 | det D1 - C1 nL)
//         last : (A4 A3 A2, det B4 - A4 B2 C3, det C4 | det D4 - A4 nR)
//     rescaled by an exact power of two; the eliminated unknowns are kept as
//         x_lL = (nL - B3 A2 x_fL + C2 C3 x_lR) / det ,   x_fR = (nR + A3 A2 x_fL - B2 C3 x_lR) / det
//     whose 1/det is computed after the merged node has been handed to the next level.
//     With m0 | m = ny/P and m/m0 a power of two, the nodes of level log2(m/m0) are exactly the
//     paper's partitions and their two equations are rows 2p, 2p+1 of its reduced system (up to
//     a row scaling).
//   * The node left per (CTA, line) is ALL-GATHERED over the cluster with asynchronous DSMEM stores
//     that complete on the receiver's mbarrier (st.async ... mbarrier::complete_tx): no cluster
//     barrier on the critical path.  Every CTA solves the 2*CL-row system with the same pairwise
//     tree and keeps its own two boundary values; then the tree is walked top-down and the leaves
//     back-substitute from registers.  Inbox and mbarrier are double-buffered by tile parity: a
//     CTA that runs ahead can only be one tile ahead (it needs everybody's tile-i data to finish
//     tile i), so its tile-(i+1) stores never land in a buffer that is still being read.
//
// Node buffer: rows 2w / 2w+1 hold the first / last equation of leaf w as 16-byte pairs (A, B) and
// (C, D); after the climb, one pass over all merges (one per thread, behind the exchange) turns the
// rows a merge eliminated into (a, c | d) of  x = d - a x_first - c x_last ; back-substitution
// overwrites D with x.  All node-buffer traffic uses explicit shared-space addresses.
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
    int max_clusters = 0;  // co-resident clusters (persistent grid size), filled at first launch
    bool xaxis = false;    // x sweep: 16-row leaves, swizzled boxes, staging tile for x
    size_t smem = 0;
};

struct TmaFusedParams {
    double *x;          // batch base of the output
    long long rs, os;   // element stride between rows of a line / between slices of the caller's
                        // arrays (y sweep: nx, nx*ny; z sweep: nx*ny, nx)
    int axis_z;         // 0: rows = tensor dim 1, slices = dim 2;  1: rows = dim 2, slices = dim 1
    int periodic;       // cyclic lines: x_{-1} = x_{n-1}, x_n = x_0 (a_0, c_{n-1} are used)
    int nx, ny, nzs;    // ny = rows per line, nzs = slices in this launch
    int CL, R, W;
    int xtiles, ntiles;
    int box_rows, nbox;
};

__host__ __device__ inline size_t tma_fused_smem_bytes(int TX, int R, int W, int CL, bool xaxis = false)
{
    if (xaxis)   // + staging tile [R][TX] for x
        return ((size_t)5 * R * TX + (size_t)4 * 2 * W * TX + (size_t)2 * 4 * 2 * CL * TX) * sizeof(double) + 128;
    // raw tile: 4 arrays [R][TX]; node buffer 4 x [2 W][TX]; cluster-level system, two inboxes of
    // 4 x [2 CL][TX]; three mbarriers (+ padding)
    return ((size_t)4 * R * TX + (size_t)4 * 2 * W * TX + (size_t)2 * 4 * 2 * CL * TX) * sizeof(double) + 128;
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

// the same for a 16-byte pair
__device__ __forceinline__ void st_async_2f64(uint32_t dst_cluster, double v0, double v1, uint32_t bar_cluster)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.b64 [%0], {%1, %2}, [%3];"
                 ::"r"(dst_cluster), "l"(__double_as_longlong(v0)), "l"(__double_as_longlong(v1)), "r"(bar_cluster)
                 : "memory");
}

}  // namespace ptx

// ------------------------------------------------------------------------------------------
// Shared-memory access by explicit 32-bit shared-space addresses (no generic-pointer arithmetic
// on the serial path), 16 bytes at a time.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ double2 lds2(uint32_t a)
{
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a));
    return v;
}
__device__ __forceinline__ double lds1(uint32_t a)
{
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ void sts2(uint32_t a, double x, double y)
{
    asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(a), "d"(x), "d"(y) : "memory");
}
__device__ __forceinline__ void sts1(uint32_t a, double x)
{
    asm volatile("st.shared.f64 [%0], %1;" ::"r"(a), "d"(x) : "memory");
}

// 2^-e for |v| in [2^e, 2^(e+1)): multiplying an equation by it is exact and brings v into [1, 2)
__device__ __forceinline__ double pow2_unscale(double v)
{
    const int e = (__double2hiint(v) >> 20) & 0x7ff;
    return __hiloint2double((2046 - e) << 20, 0);
}

// Branch-free reciprocal: hardware seed (MUFU.RCP64H, ~2^-20) + two Newton steps, within about
// one ulp.  Unlike 1.0 / x it has no slow-path branch, so independent recurrences interleave in
// one basic block.  Valid for normal, non-huge |x| (2^-1021 < |x| < 2^1021); x = 0 gives inf.
__device__ __forceinline__ double rcp_nr(double x)
{
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    double e = fma(-x, r, 1.0);
    r = fma(r, e, r);
    e = fma(-x, r, 1.0);
    return fma(r, e, r);
}

struct Eq { double a, b, c, d; };

// Node buffer: `rows` equations x TX lines, stored as two planes of 16-byte pairs,
//   AB[row][line] = (A, B)   and   CD[row][line] = (C, D),   CD plane `plane` bytes after AB.
// An eliminated row keeps (a, c) in its AB slot and d (later x) in the D half of its CD slot.
struct NodeBuf { uint32_t ab, plane; };

template <int TX>
__device__ __forceinline__ uint32_t nb_ab(const NodeBuf &nb, int row, int lx) { return nb.ab + (uint32_t)(row * TX + lx) * 16u; }

// Pairwise merge, first half (see the header): rows r1 < r2 < r3 < r4 hold L.first, L.last,
// R.first, R.last; r1 / r4 receive the merged node's equations.  Division-free.
template <int TX>
__device__ __forceinline__ void merge_head(const NodeBuf &nb, int lx, int r1, int r2, int r3, int r4)
{
    const uint32_t o1 = nb_ab<TX>(nb, r1, lx), o2 = nb_ab<TX>(nb, r2, lx), o3 = nb_ab<TX>(nb, r3, lx), o4 = nb_ab<TX>(nb, r4, lx);
    const double2 ab2 = lds2(o2), cd2 = lds2(o2 + nb.plane), ab3 = lds2(o3), cd3 = lds2(o3 + nb.plane);
    const double2 ab1 = lds2(o1), cd1 = lds2(o1 + nb.plane), ab4 = lds2(o4), cd4 = lds2(o4 + nb.plane);
    const double A2 = ab2.x, B2 = ab2.y, C2 = cd2.x, D2 = cd2.y, A3 = ab3.x, B3 = ab3.y, C3 = cd3.x, D3 = cd3.y;
    const double A1 = ab1.x, B1 = ab1.y, C1 = cd1.x, D1 = cd1.y, A4 = ab4.x, B4 = ab4.y, C4 = cd4.x, D4 = cd4.y;
    const double det = fma(B2, B3, -(C2 * A3));
    const double nL = fma(B3, D2, -(C2 * D3)), nR = fma(B2, D3, -(A3 * D2));
    const double p1 = B3 * A2, p2 = C2 * C3, p3 = A3 * A2, p4 = B2 * C3;
    double fb = fma(det, B1, -(C1 * p1)), lb = fma(det, B4, -(A4 * p4));
    const double sf = pow2_unscale(fb), sl = pow2_unscale(lb);
    sts2(o1, det * A1 * sf, fb * sf);
    sts2(o1 + nb.plane, C1 * p2 * sf, fma(det, D1, -(C1 * nL)) * sf);
    sts2(o4, A4 * p3 * sl, lb * sl);
    sts2(o4 + nb.plane, det * C4 * sl, fma(det, D4, -(A4 * nR)) * sl);
}

// Second half, recomputed from the two rows the merge eliminated (they are untouched until now):
// x_lL = d - a x_first - c x_last in row r2, x_fR likewise in row r3.
template <int TX>
__device__ __forceinline__ void merge_tail(const NodeBuf &nb, int lx, int r2, int r3)
{
    const uint32_t o2 = nb_ab<TX>(nb, r2, lx), o3 = nb_ab<TX>(nb, r3, lx);
    const double2 ab2 = lds2(o2), cd2 = lds2(o2 + nb.plane), ab3 = lds2(o3), cd3 = lds2(o3 + nb.plane);
    const double A2 = ab2.x, B2 = ab2.y, C2 = cd2.x, D2 = cd2.y, A3 = ab3.x, B3 = ab3.y, C3 = cd3.x, D3 = cd3.y;
    const double inv = rcp_nr(fma(B2, B3, -(C2 * A3)));
    const double nL = fma(B3, D2, -(C2 * D3)), nR = fma(B2, D3, -(A3 * D2));
    sts2(o2, (B3 * A2) * inv, -((C2 * C3) * inv));
    sts1(o2 + nb.plane + 8, nL * inv);
    sts2(o3, -((A3 * A2) * inv), (B2 * C3) * inv);
    sts1(o3 + nb.plane + 8, nR * inv);
}

template <int TX>
__device__ __forceinline__ void unmerge_pair(const NodeBuf &nb, int lx, int r1, int r2, int r3, int r4)
{
    const uint32_t o2 = nb_ab<TX>(nb, r2, lx), o3 = nb_ab<TX>(nb, r3, lx);
    const double xf = lds1(nb_ab<TX>(nb, r1, lx) + nb.plane + 8), xl = lds1(nb_ab<TX>(nb, r4, lx) + nb.plane + 8);
    const double2 ac2 = lds2(o2), ac3 = lds2(o3);
    const double d2 = lds1(o2 + nb.plane + 8), d3 = lds1(o3 + nb.plane + 8);
    sts1(o2 + nb.plane + 8, fma(-ac2.y, xl, fma(-ac2.x, xf, d2)));
    sts1(o3 + nb.plane + 8, fma(-ac3.y, xl, fma(-ac3.x, xf, d3)));
}

// Pairwise tree over `nodes` nodes (a power of two) of 2 rows each, one line per lx, thread rows
// `slot` of `nslots`.  Bottom-up, heads only: on return (after its closing __syncthreads) the root
// has its first equation in row 0 and its last equation in row 2*nodes-1.
template <int TX>
__device__ __forceinline__ void tree_up(const NodeBuf &nb, int lx, int slot, int nslots, int nodes,
                                        bool synced = false)
{
    for (int n = nodes, sp = 2; n > 1; n >>= 1, sp <<= 1) {
        if (!(synced && n == nodes)) __syncthreads();   // synced: the caller has just done the first one
        for (int q = slot; q < (n >> 1); q += nslots) {
            const int rs = q * 2 * sp;
            merge_head<TX>(nb, lx, rs, rs + sp - 1, rs + sp, rs + 2 * sp - 1);
        }
    }
    __syncthreads();
}

// The tails of ALL merges of tree_up, one per thread row: merge j of the flat list (level 1 pairs,
// then level 2 pairs, ...) goes to slot j.  No barrier inside; needs one before tree_down.
template <int TX>
__device__ __forceinline__ void tree_tails(const NodeBuf &nb, int lx, int slot, int nslots, int nodes)
{
    for (int j = slot; j < nodes - 1; j += nslots) {
        int base = 0, n = nodes, sp = 2;
        while (j - base >= (n >> 1)) { base += n >> 1; n >>= 1; sp <<= 1; }
        const int rs = (j - base) * 2 * sp;
        merge_tail<TX>(nb, lx, rs + sp - 1, rs + sp);
    }
}

// Top-down: needs x_first / x_last of the root in D of row 0 / row 2*nodes-1 and all tails
// (visible to all threads); ends with a __syncthreads().
template <int TX>
__device__ __forceinline__ void tree_down(const NodeBuf &nb, int lx, int slot, int nslots, int nodes)
{
    for (int n = 2, sp = nodes; n <= nodes; n <<= 1, sp >>= 1) {
        for (int q = slot; q < (n >> 1); q += nslots) {
            const int rs = q * 2 * sp;
            unmerge_pair<TX>(nb, lx, rs, rs + sp - 1, rs + sp, rs + 2 * sp - 1);
        }
        __syncthreads();
    }
}

// Root of a tree: first equation  A x_prev + B x_f + C x_l = D  (row 0), last equation
// A x_f + B x_l + C x_next = D  (row rl)  ->  x_f, x_l into D.  Plain lines: the root's A_first and
// C_last are 0.  Cyclic lines (wrap): x_prev = x_l and x_next = x_f, i.e. the periodic coupling is
// resolved here, at the top of the recursion, as  B_f x_f + (A_f + C_f) x_l = D_f ,
// (A_l + C_l) x_f + B_l x_l = D_l  -- no Sherman-Morrison correction is needed.
template <int TX>
__device__ __forceinline__ void solve_root(const NodeBuf &nb, int lx, int rl, bool wrap)
{
    const uint32_t oF = nb_ab<TX>(nb, 0, lx), oL = nb_ab<TX>(nb, rl, lx);
    const double2 abf = lds2(oF), cdf = lds2(oF + nb.plane), abl = lds2(oL), cdl = lds2(oL + nb.plane);
    const double Cf = wrap ? cdf.x + abf.x : cdf.x, Al = wrap ? abl.x + cdl.x : abl.x;
    const double inv = rcp_nr(fma(abf.y, abl.y, -(Cf * Al)));
    sts1(oL + nb.plane + 8, fma(abf.y, cdl.y, -(Al * cdf.y)) * inv);
    sts1(oF + nb.plane + 8, fma(abl.y, cdf.y, -(Cf * cdl.y)) * inv);
}

// Leaf state of one thread: M0 rows of one line, swept as K = M0/H independent sub-leaves of H rows
// (two interleaved recurrences when M0 >= 8) that are merged in registers.  What stays in
// registers until back-substitution: the interior rows of every sub-leaf, (ia, ic, id) of
// x_r = id - ia x_first - ic x_{r+1}, and for K = 2 the two unknowns the in-register merge
// eliminated, (ma, mc, md)[j] of x = md - ma x_0 - mc x_{M0-1}  (j = 0: row H-1, j = 1: row H).
template <int M0>
struct LeafRegs {
    static constexpr int K = M0 >= 8 ? 2 : 1;
    static constexpr int H = M0 / K;
    static constexpr int HI = H > 2 ? H - 2 : 1;
    double ia[K][HI], ic[K][HI], id[K][HI];
    double ma[2], mc[2], md[2];
};

// Last step of a leaf sweep: normalise the first-row equations of the sub-leaves and, for two
// sub-leaves, merge them pairwise in registers.
template <int M0>
__device__ __forceinline__ void leaf_finish(double (&fa)[LeafRegs<M0>::K], double (&fb)[LeafRegs<M0>::K],
                                            double (&fc)[LeafRegs<M0>::K], double (&fd)[LeafRegs<M0>::K],
                                            double (&pa)[LeafRegs<M0>::K], double (&pc)[LeafRegs<M0>::K],
                                            double (&pd)[LeafRegs<M0>::K], Eq &f, Eq &l, LeafRegs<M0> &R)
{
    constexpr int K = LeafRegs<M0>::K;
#pragma unroll
    for (int h = 0; h < K; ++h) {                                // H == 2: fb = 1, frontier is x_1
        const double inv = rcp_nr(fb[h]);
        fa[h] *= inv; fc[h] *= inv; fd[h] *= inv;
    }
    if (K == 1) {
        f.a = fa[0]; f.b = 1.0; f.c = fc[0]; f.d = fd[0];
        l.a = pa[0]; l.b = 1.0; l.c = pc[0]; l.d = pd[0];
    } else {
        // pairwise merge of the two sub-leaves in registers (unit diagonals):
        // (A1, C1, D1) = first / (A2, C2, D2) = last eq of sub-leaf 0, (A3..), (A4..) of sub-leaf 1
        const double A1 = fa[0], C1 = fc[0], D1 = fd[0], A2 = pa[0], C2 = pc[0], D2 = pd[0];
        const double A3 = fa[K - 1], C3 = fc[K - 1], D3 = fd[K - 1], A4 = pa[K - 1], C4 = pc[K - 1], D4 = pd[K - 1];
        const double det = fma(-C2, A3, 1.0);
        const double nL = fma(-C2, D3, D2), nR = fma(-A3, D2, D3);
        const double p2 = C2 * C3, p3 = A3 * A2;
        f.b = fma(-C1, A2, det); l.b = fma(-A4, C3, det);
        const double sf = pow2_unscale(f.b), sl = pow2_unscale(l.b);
        f.a = det * A1 * sf; f.b *= sf; f.c = C1 * p2 * sf; f.d = fma(det, D1, -(C1 * nL)) * sf;
        l.a = A4 * p3 * sl; l.b *= sl; l.c = det * C4 * sl; l.d = fma(det, D4, -(A4 * nR)) * sl;
        const double inv = rcp_nr(det);
        R.ma[0] = A2 * inv; R.mc[0] = -(p2 * inv); R.md[0] = nL * inv;
        R.ma[1] = -(p3 * inv); R.mc[1] = C3 * inv; R.md[1] = nR * inv;
    }
}

// Modified Thomas reduction (tdma_stage_kernels.cuh) of the sub-leaves, read from the raw tile at
// offset o0 (row stride TX).  Returns the leaf's two boundary equations
//   f: A x_prev + B x_0 + C x_last = D        l: A x_0 + B x_last + C x_next = D
template <int TX, int M0>
__device__ __forceinline__ void leaf_reduce(const double *__restrict__ sA, const double *__restrict__ sB,
                                            const double *__restrict__ sC, const double *__restrict__ sD,
                                            int o0, bool first_leaf, bool last_leaf, Eq &f, Eq &l,
                                            LeafRegs<M0> &R)
{
    constexpr int K = LeafRegs<M0>::K, H = LeafRegs<M0>::H;
    double fa[K], fb[K], fc[K], fd[K], pa[K], pc[K], pd[K];
#pragma unroll
    for (int h = 0; h < K; ++h) {
        const int o = o0 + h * H * TX;
        double inv = rcp_nr(sB[o]);
        fa[h] = (h == 0 && first_leaf) ? 0.0 : sA[o] * inv;      // global a_0 := 0
        fc[h] = sC[o] * inv;
        fd[h] = sD[o] * inv;
        fb[h] = 1.0;
        double c1 = sC[o + TX];
        if (H == 2 && h == K - 1 && last_leaf) c1 = 0.0;         // global c_{ny-1} := 0
        inv = rcp_nr(sB[o + TX]);
        pa[h] = sA[o + TX] * inv; pc[h] = c1 * inv; pd[h] = sD[o + TX] * inv;
    }
#pragma unroll
    for (int r = 2; r < H; ++r) {
#pragma unroll
        for (int h = 0; h < K; ++h) {
            const int o = o0 + (h * H + r) * TX;
            const double ar = sA[o], br = sB[o], dr = sD[o];
            double cr = sC[o];
            if (r == H - 1 && h == K - 1 && last_leaf) cr = 0.0;
            // fold row r-1 into the first-row equation, park it for back-substitution
            fb[h] = fma(-fc[h], pa[h], fb[h]);
            fd[h] = fma(-fc[h], pd[h], fd[h]);
            fc[h] = -fc[h] * pc[h];
            R.ia[h][r - 2] = pa[h]; R.ic[h][r - 2] = pc[h]; R.id[h][r - 2] = pd[h];
            const double inv = rcp_nr(fma(-ar, pc[h], br));
            pd[h] = fma(-ar, pd[h], dr) * inv;
            pc[h] = cr * inv;
            pa[h] = -(ar * pa[h]) * inv;
        }
    }
    leaf_finish<M0>(fa, fb, fc, fd, pa, pc, pd, f, l, R);
}

// Back-substitution of the leaf from registers given its first and last unknown; x streamed to
// HBM (row stride nx elements).
template <int M0>
__device__ __forceinline__ void leaf_back(const LeafRegs<M0> &R, double xf, double xl, double *__restrict__ xp,
                                          size_t nx)
{
    constexpr int K = LeafRegs<M0>::K, H = LeafRegs<M0>::H;
    double first[K], last[K];
    first[0] = xf; last[K - 1] = xl;
    if (K == 2) {
        last[0] = fma(-R.mc[0], xl, fma(-R.ma[0], xf, R.md[0]));
        first[K - 1] = fma(-R.mc[1], xl, fma(-R.ma[1], xf, R.md[1]));
    }
    double xn[K];
#pragma unroll
    for (int h = 0; h < K; ++h) {
        xn[h] = last[h];
        __stcs(xp + (size_t)(h * H) * nx, first[h]);
        __stcs(xp + (size_t)(h * H + H - 1) * nx, last[h]);
    }
#pragma unroll
    for (int r = H - 2; r >= 1; --r) {
#pragma unroll
        for (int h = 0; h < K; ++h) {
            xn[h] = fma(-R.ic[h][r - 1], xn[h], fma(-R.ia[h][r - 1], first[h], R.id[h][r - 1]));
            __stcs(xp + (size_t)(h * H + r) * nx, xn[h]);
        }
    }
}

// ------------------------------------------------------------------------------------------
// x sweeps (lines along the fastest axis).  A leaf is 16 consecutive x of one line = one 128-byte
// row; the raw tile arrives as one (16 x, TX lines) TMA box per leaf and array with the 128-byte
// swizzle: the 16-byte chunk q of box row l sits at chunk q ^ (l & 7).  A thread reads its row
// with 16-byte loads; the 8 lanes of a quarter warp (8 consecutive lines) then touch 8 different
// chunks, i.e. all 32 banks once.  x goes back through a staging tile with the same layout and
// one TMA store per leaf box.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t xs_addr(uint32_t box, int l, int pair)
{
    return box + (uint32_t)l * 128u + (uint32_t)((pair ^ (l & 7)) << 4);
}

// bA..bD: shared addresses of this leaf's boxes.  Same arithmetic as leaf_reduce<TX, 16>.
__device__ __forceinline__ void leaf_reduce_x(uint32_t bA, uint32_t bB, uint32_t bC, uint32_t bD, int l,
                                              bool first_leaf, bool last_leaf, Eq &f, Eq &le, LeafRegs<16> &R)
{
    constexpr int K = 2, H = 8;
    double fa[K], fb[K], fc[K], fd[K], pa[K], pc[K], pd[K];
#pragma unroll
    for (int h = 0; h < K; ++h) {
        const double2 a2 = lds2(xs_addr(bA, l, 4 * h)), b2 = lds2(xs_addr(bB, l, 4 * h));
        const double2 c2 = lds2(xs_addr(bC, l, 4 * h)), d2 = lds2(xs_addr(bD, l, 4 * h));
        double inv = rcp_nr(b2.x);
        fa[h] = (h == 0 && first_leaf) ? 0.0 : a2.x * inv;
        fc[h] = c2.x * inv; fd[h] = d2.x * inv; fb[h] = 1.0;
        inv = rcp_nr(b2.y);
        pa[h] = a2.y * inv; pc[h] = c2.y * inv; pd[h] = d2.y * inv;
    }
#pragma unroll
    for (int p = 1; p < H / 2; ++p) {
        double2 a2[K], b2[K], c2[K], d2[K];
#pragma unroll
        for (int h = 0; h < K; ++h) {
            a2[h] = lds2(xs_addr(bA, l, 4 * h + p)); b2[h] = lds2(xs_addr(bB, l, 4 * h + p));
            c2[h] = lds2(xs_addr(bC, l, 4 * h + p)); d2[h] = lds2(xs_addr(bD, l, 4 * h + p));
        }
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const int r = 2 * p + e;
#pragma unroll
            for (int h = 0; h < K; ++h) {
                const double ar = e ? a2[h].y : a2[h].x, br = e ? b2[h].y : b2[h].x, dr = e ? d2[h].y : d2[h].x;
                double cr = e ? c2[h].y : c2[h].x;
                if (r == H - 1 && h == K - 1 && last_leaf) cr = 0.0;
                fb[h] = fma(-fc[h], pa[h], fb[h]);
                fd[h] = fma(-fc[h], pd[h], fd[h]);
                fc[h] = -fc[h] * pc[h];
                R.ia[h][r - 2] = pa[h]; R.ic[h][r - 2] = pc[h]; R.id[h][r - 2] = pd[h];
                const double inv = rcp_nr(fma(-ar, pc[h], br));
                pd[h] = fma(-ar, pd[h], dr) * inv;
                pc[h] = cr * inv;
                pa[h] = -(ar * pa[h]) * inv;
            }
        }
    }
    leaf_finish<16>(fa, fb, fc, fd, pa, pc, pd, f, le, R);
}

// Back-substitution of a 16-row leaf into the staging box bX (row l).
__device__ __forceinline__ void leaf_back_x(const LeafRegs<16> &R, double xf, double xl, uint32_t bX, int l)
{
    constexpr int K = 2, H = 8;
    double xs[16];
    double first[K], last[K];
    first[0] = xf; last[1] = xl;
    last[0] = fma(-R.mc[0], xl, fma(-R.ma[0], xf, R.md[0]));
    first[1] = fma(-R.mc[1], xl, fma(-R.ma[1], xf, R.md[1]));
#pragma unroll
    for (int h = 0; h < K; ++h) {
        xs[h * H] = first[h]; xs[h * H + H - 1] = last[h];
        double xn = last[h];
#pragma unroll
        for (int r = H - 2; r >= 1; --r) {
            xn = fma(-R.ic[h][r - 1], xn, fma(-R.ia[h][r - 1], first[h], R.id[h][r - 1]));
            xs[h * H + r] = xn;
        }
    }
#pragma unroll
    for (int p = 0; p < 8; ++p) sts2(xs_addr(bX, l, p), xs[2 * p], xs[2 * p + 1]);
}

// kX: x sweep (lanes = TX lines along y, rows = x; M0 = 16 only); tm_x is used by x sweeps only.
template <int TX, int M0, bool kCluster, int MAXT, int MINB, bool kX>
__global__ void __launch_bounds__(MAXT, MINB)
fused_tma_kernel(const __grid_constant__ CUtensorMap tm_a, const __grid_constant__ CUtensorMap tm_b,
                 const __grid_constant__ CUtensorMap tm_c, const __grid_constant__ CUtensorMap tm_d,
                 const __grid_constant__ CUtensorMap tm_x, const TmaFusedParams prm)
{
    static_assert(!kX || M0 == 16, "x sweeps use 16-row (128-byte) leaves");
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    const int R = prm.R, CL = prm.CL, W = prm.W;
    const int arr = R * TX;
    double *__restrict__ sA = reinterpret_cast<double *>(smem_raw);   // raw tile
    double *__restrict__ sB = sA + arr;
    double *__restrict__ sC = sB + arr;
    double *__restrict__ sD = sC + arr;
    const int narr = 2 * W * TX;
    double *sX = sD + arr;                                            // x staging tile (x sweeps)
    double *node = sX + (kX ? arr : 0);                               // node buffer, 4 x [2W][TX]
    const int NTR = 2 * CL;                                    // rows of the cluster-level system
    const int tarr = NTR * TX;
    double *top = node + 4 * narr;                             // 2 inboxes x 4 x [NTR][TX]
    uint64_t *bar = reinterpret_cast<uint64_t *>(top + 8 * tarr);   // [0]: raw tile, [1], [2]: inboxes
    NodeBuf nb;
    nb.ab = ptx::smem_u32(node); nb.plane = (uint32_t)narr * 16u;

    const int t = threadIdx.x;
    unsigned crank = 0;
    if (kCluster) crank = cg::this_cluster().block_rank();
    const int g = blockIdx.x / CL, NC = gridDim.x / CL;        // cluster index / number of clusters
    const int lx = t % TX, leaf = t / TX;
    const int y0 = (int)crank * R;
    const int o0 = leaf * M0 * TX + lx;
    const bool first_leaf = !prm.periodic && (y0 + leaf * M0 == 0);
    const bool last_leaf = !prm.periodic && (y0 + leaf * M0 + M0 == prm.ny);

    // The whole raw tile of `tile` in flight at once.  One copy costs its issuing thread 150-200
    // cycles (measured), so inside the loop the four arrays are issued by lane 0 of four DIFFERENT
    // warps -- the last four, which have no merge to do at the first tree level -- and the climb
    // does not wait for them.  sel < 0: all arrays (prologue); sel = 0..3: array sel only.
    auto issue_tile = [&](int tile, int sel) {
        const int x0 = (tile % prm.xtiles) * TX, k = tile / prm.xtiles;
        if (sel <= 0) ptx::mbar_expect_tx(&bar[0], (unsigned)(4 * arr * sizeof(double)));
        double *const dst[4] = {sB, sA, sC, sD};
        const CUtensorMap *const tm[4] = {&tm_b, &tm_a, &tm_c, &tm_d};
        for (int a = 0; a < 4; ++a) {
            if (sel >= 0 && sel != a) continue;
            if (kX) {                   // one (16 x, TX lines) box per leaf; x0 = first line (y)
                for (int w = 0; w < W; ++w)
                    ptx::tma_load_3d(dst[a] + w * 16 * TX, tm[a], y0 + 16 * w, x0, k, &bar[0]);
            } else for (int q = 0; q < prm.nbox; ++q) {
                const int yy = y0 + q * prm.box_rows;
                const int c1 = prm.axis_z ? k : yy, c2 = prm.axis_z ? yy : k;
                ptx::tma_load_3d(dst[a] + q * prm.box_rows * TX, tm[a], x0, c1, c2, &bar[0]);
            }
        }
    };
    const int nwarps = ((int)blockDim.x + 31) / 32;
    // my role in the in-loop issue: -1 none, -2 everything (CTAs with fewer than 8 warps), 0..3 array
    const int issue_sel = nwarps >= 8 ? (((t & 31) == 0 && t / 32 >= nwarps - 4) ? t / 32 - (nwarps - 4) : -1)
                                      : (t == 0 ? -2 : -1);

    if (t == 0) {
        ptx::mbar_init(&bar[0], 1);
        ptx::mbar_init(&bar[1], 1);
        ptx::mbar_init(&bar[2], 1);
        ptx::fence_mbar_init();
        issue_tile(g, -1);
    }
    __syncthreads();                    // mbarriers initialised before anyone waits on them
    // split-phase cluster barrier: "every CTA of the cluster has started and initialised its
    // inbox mbarriers" must hold before the first remote store; the matching wait sits right
    // before the first exchange, where it is satisfied long ago
    if (kCluster) asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");

    int it = 0;
    for (int tile = g; tile < prm.ntiles; tile += NC, ++it) {
        const int par = it & 1;
        NodeBuf tb;                                            // this tile's inbox
        tb.ab = ptx::smem_u32(top + par * 4 * tarr); tb.plane = (uint32_t)tarr * 16u;
        // arm this tile's inbox: 4 doubles per (node equation, line) from every CTA
        if (kCluster && t == 0) ptx::mbar_expect_tx(&bar[1 + par], (unsigned)(4 * tarr * sizeof(double)));
        if (kX && t == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
        ptx::mbar_wait(&bar[0], (unsigned)par);

        // ---------------- leaves ----------------
        LeafRegs<M0> regs;
        {
            Eq f, l;
            if constexpr (kX) {
                const uint32_t bo = (uint32_t)(leaf * 16 * TX) * 8u;
                leaf_reduce_x(ptx::smem_u32(sA) + bo, ptx::smem_u32(sB) + bo, ptx::smem_u32(sC) + bo,
                              ptx::smem_u32(sD) + bo, lx, first_leaf, last_leaf, f, l, regs);
            } else {
                leaf_reduce<TX, M0>(sA, sB, sC, sD, o0, first_leaf, last_leaf, f, l, regs);
            }
            const uint32_t of = nb_ab<TX>(nb, 2 * leaf, lx), ol = of + TX * 16u;
            sts2(of, f.a, f.b); sts2(of + nb.plane, f.c, f.d);
            sts2(ol, l.a, l.b); sts2(ol + nb.plane, l.c, l.d);
        }
        __syncthreads();                // raw tile consumed, node equations visible
        if (issue_sel != -1 && tile + NC < prm.ntiles) issue_tile(tile + NC, issue_sel == -2 ? -1 : issue_sel);   // prefetch behind the tree

        // ---------------- pairwise tree inside the CTA, bottom-up ----------------
        tree_up<TX>(nb, lx, leaf, W, W, true);

        // ---------------- cluster level ----------------
        // the CTA's node: first equation in node row 0, last equation in node row 2W-1
        if (!kCluster) {
            if (t < TX) solve_root<TX>(nb, lx, 2 * W - 1, prm.periodic != 0);
            tree_tails<TX>(nb, lx, leaf, W, W);
            __syncthreads();
        } else {
            // A2B as an all-gather (the paper's MPI_Alltoall, with every rank
            // keeping a copy): asynchronous DSMEM stores that complete on the RECEIVER's mbarrier
            if (it == 0) asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
            const uint32_t bar_s = ptx::smem_u32(&bar[1 + par]);
            for (int e = t; e < 2 * TX * CL; e += (int)blockDim.x) {
                const int dest = e / (2 * TX), r = e - dest * 2 * TX;
                const int j = r / TX, l = r - j * TX;      // j: 0 = first eq, 1 = last eq
                const uint32_t src = nb_ab<TX>(nb, j ? 2 * W - 1 : 0, l);
                const double2 ab = lds2(src), cd = lds2(src + nb.plane);
                const uint32_t dst = ptx::mapa(nb_ab<TX>(tb, (int)crank * 2 + j, l), (unsigned)dest);
                const uint32_t dbar = ptx::mapa(bar_s, (unsigned)dest);
                ptx::st_async_2f64(dst, ab.x, ab.y, dbar);
                ptx::st_async_2f64(dst + tb.plane, cd.x, cd.y, dbar);
            }
            // the reciprocals of the tree just climbed run behind the exchange
            tree_tails<TX>(nb, lx, leaf, W, W);
            ptx::mbar_wait(&bar[1 + par], (unsigned)((it >> 1) & 1));
            // Stage B: the 2*CL-row system, solved redundantly by every CTA with the same
            // pairwise tree, so no second exchange is needed
            tree_up<TX>(tb, lx, leaf, W, CL);
            if (t < TX) solve_root<TX>(tb, lx, NTR - 1, prm.periodic != 0);
            tree_tails<TX>(tb, lx, leaf, W, CL);
            __syncthreads();
            tree_down<TX>(tb, lx, leaf, W, CL);
            // B2C: my node's boundary values
            for (int e = t; e < 2 * TX; e += (int)blockDim.x) {
                const int j = e / TX, l = e - j * TX;
                sts1(nb_ab<TX>(nb, j ? 2 * W - 1 : 0, l) + nb.plane + 8,
                     lds1(nb_ab<TX>(tb, (int)crank * 2 + j, l) + tb.plane + 8));
            }
            __syncthreads();
        }

        // ---------------- pairwise tree inside the CTA, top-down ----------------
        tree_down<TX>(nb, lx, leaf, W, W);

        // ---------------- leaves: back-substitution from registers, x streamed to HBM --------
        {
            const int x0 = (tile % prm.xtiles) * TX, k = tile / prm.xtiles;
            const double xf = lds1(nb_ab<TX>(nb, 2 * leaf, lx) + nb.plane + 8);
            const double xl = lds1(nb_ab<TX>(nb, 2 * leaf + 1, lx) + nb.plane + 8);
            if constexpr (kX) {
                // the staging tile of the previous iteration has been read by the TMA engine
                // (thread 0 waited at the top of this iteration, barriers in between)
                leaf_back_x(regs, xf, xl, ptx::smem_u32(sX) + (uint32_t)(leaf * 16 * TX) * 8u, lx);
                ptx::fence_proxy_async_smem();
                __syncthreads();
                if (t == 0) {
                    for (int w = 0; w < W; ++w)
                        ptx::tma_store_3d(&tm_x, y0 + 16 * w, x0, k, sX + w * 16 * TX);
                    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
                }
            } else if (x0 + lx < prm.nx) {     // ragged last x tile: TMA zero-filled those lanes
                leaf_back<M0>(regs, xf, xl,
                              prm.x + (size_t)k * (size_t)prm.os + (size_t)(y0 + leaf * M0) * (size_t)prm.rs +
                                  (size_t)(x0 + lx), (size_t)prm.rs);
            }
        }
    }
    // the staging tile must outlive the last TMA store
    if (kX && t == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
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
                                const char **why, bool xaxis = false, bool zaxis = false)
{
    // x sweep: nx = number of lanes (caller's ny), ny = line length (caller's nx)
    if (xaxis) {
        if (ny % 2) { *why = "TMA path needs even nx (16-byte global strides)"; return false; }
        if ((want_lines && want_lines != 16) || (want_leaf && want_leaf != 16)) {
            *why = "x sweeps use 16 lines per tile and 16-row leaves"; return false;
        }
        want_lines = 16; want_leaf = 16;
    } else if (nx % 2) { *why = "TMA path needs even nx (16-byte global strides)"; return false; }
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
                if (c.threads > 1024 || (xaxis && c.threads > 256)) continue;
                c.nlev = 0;
                while ((1 << c.nlev) < c.leaves) ++c.nlev;
                c.box_rows = R;
                while (c.box_rows > 256) c.box_rows /= 2;
                if (R % c.box_rows) continue;
                c.xaxis = xaxis;
                c.smem = tma_fused_smem_bytes(TX, R, c.leaves, CL, xaxis);
                if (c.smem > max_smem) continue;
                long ctas = (long)(sm_smem / (c.smem + 1024));
                const long by_thr = 2048 / c.threads;
                if (by_thr < ctas) ctas = by_thr;
                if (ctas < 1) continue;
                // Measured on B200 (cfg 3 shapes): the tile period is set by the serial phases, so
                // long leaves (fewer tree levels) win first; then two CTAs per SM (one sweeps while
                // the other walks its tree), resident cells, small clusters, 64-128 B row segments.
                // registers per thread of the instantiation (see launch_tma_m0)
                const long regs = c.threads > 512 ? 64 : (c.threads > 256 || m0 < 16 ? 128 : 256);
                const long by_regs = 65536 / (regs * c.threads);
                if (by_regs < ctas) ctas = by_regs;
                if (ctas < 1) continue;
                double cells = (double)ctas * R * TX;
                if (cells > 8192.0) cells = 8192.0;
                // 128 B row segments: with 64 B segments the persistent clusters drift apart in a
                // long run and DRAM row-buffer locality between neighbouring x tiles is lost
                // (measured: 4.4 -> 3.1 TB/s from 256 to 1024 slices at TX = 8, flat at TX = 16)
                double score = 10000.0 * m0 + cells + (c.threads >= 32 ? 4000.0 : 0.0) + (ctas >= 2 ? 100.0 : 0.0) -
                               50.0 * CL +
                               // z sweeps: rows of a line are whole slices apart (a DRAM page and a
                               // TLB entry per row), 256 B segments pay (0.99 -> 0.91 ms on cfg 4)
                               (zaxis ? (TX == 32 ? 3000.0 : (TX == 16 ? 1000.0 : 0.0))
                                      : (TX == 16 ? 3000.0 : (TX == 32 ? 1000.0 : 0.0)));
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

// fp64 slab with x fastest; rows of a line rs elements apart, slices os elements apart.
// y sweep: tensor (nx, rows, slices), box (TX, box_rows, 1); z sweep: tensor (nx, slices, rows),
// box (TX, 1, box_rows) -- either way the box lands in shared memory as [box_rows][TX].
inline bool make_slab_tensor_map(CUtensorMap *tm, const void *base, int nx, int nrows, int nslices,
                                 long long rs, long long os, bool axis_z, int TX, int box_rows)
{
    tdma_encode_tiled_fn enc = get_encode_tiled();
    if (!enc) return false;
    cuuint64_t gdim[3] = {(cuuint64_t)nx, (cuuint64_t)(axis_z ? nslices : nrows), (cuuint64_t)(axis_z ? nrows : nslices)};
    cuuint64_t gstr[2] = {(cuuint64_t)(axis_z ? os : rs) * sizeof(double), (cuuint64_t)(axis_z ? rs : os) * sizeof(double)};
    cuuint32_t box[3] = {(cuuint32_t)TX, (cuuint32_t)(axis_z ? 1 : box_rows), (cuuint32_t)(axis_z ? box_rows : 1)};
    cuuint32_t estr[3] = {1, 1, 1};
    const size_t inner = (size_t)TX * sizeof(double);   // one L2 request per row segment, no over-fetch
    const CUtensorMapL2promotion promo = inner >= 256 ? CU_TENSOR_MAP_L2_PROMOTION_L2_256B
                                       : inner >= 128 ? CU_TENSOR_MAP_L2_PROMOTION_L2_128B
                                                      : CU_TENSOR_MAP_L2_PROMOTION_L2_64B;
    return enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<void *>(base), gdim, gstr, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, promo,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// x sweep: contiguous fp64 slab (rows = x fastest, lanes = y, slices); box (16 x, TX lanes, 1)
// with the 128-byte swizzle.
inline bool make_xsweep_tensor_map(CUtensorMap *tm, const void *base, int nrows, int nlanes, int nslices, int TX)
{
    tdma_encode_tiled_fn enc = get_encode_tiled();
    if (!enc) return false;
    cuuint64_t gdim[3] = {(cuuint64_t)nrows, (cuuint64_t)nlanes, (cuuint64_t)nslices};
    cuuint64_t gstr[2] = {(cuuint64_t)nrows * sizeof(double), (cuuint64_t)nrows * nlanes * sizeof(double)};
    cuuint32_t box[3] = {16, (cuuint32_t)TX, 1};
    cuuint32_t estr[3] = {1, 1, 1};
    return enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<void *>(base), gdim, gstr, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int TX, int M0, bool kCluster, int MAXT, int MINB, bool kX = false>
inline cudaError_t launch_tma_inst(TmaFusedConfig &cfg, const CUtensorMap *tm, const TmaFusedParams &prm,
                                   cudaStream_t st)
{
    auto kern = fused_tma_kernel<TX, M0, kCluster, MAXT, MINB, kX>;
    size_t smem_bytes = cfg.smem;
    cudaLaunchConfig_t lc = {};
    lc.blockDim = dim3(cfg.threads);
    lc.dynamicSmemBytes = smem_bytes;
    lc.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = cfg.cluster; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    lc.attrs = attr;
    lc.numAttrs = kCluster ? 1 : 0;
    if (cfg.max_clusters <= 0) {        // first launch of this plan: attributes + persistent grid size
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes);
        if (e != cudaSuccess) return e;
        if (cfg.cluster > 8) {
            e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
            if (e != cudaSuccess) return e;
        }
        int dev = 0, sms = 0, n = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (kCluster) {
            lc.gridDim = dim3((unsigned)(cfg.cluster * sms));
            e = cudaOccupancyMaxActiveClusters(&n, kern, &lc);
            if (e != cudaSuccess) return e;
        } else {
            e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kern, cfg.threads, smem_bytes);
            if (e != cudaSuccess) return e;
            n *= sms;
        }
        if (n < 1) return cudaErrorLaunchOutOfResources;
        cfg.max_clusters = n;
    }
    if (prm.ntiles <= 0) return cudaSuccess;    // prepare only (attributes + persistent grid size)
    const int nc = prm.ntiles < cfg.max_clusters ? prm.ntiles : cfg.max_clusters;
    lc.gridDim = dim3((unsigned)(nc * cfg.cluster));
    return cudaLaunchKernelEx(&lc, kern, tm[0], tm[1], tm[2], tm[3], tm[4], prm);
}

template <int TX, int M0, bool kCluster>
inline cudaError_t launch_tma_m0(TmaFusedConfig &cfg, const CUtensorMap *tm, const TmaFusedParams &prm,
                                 cudaStream_t st)
{
    // registers: the parked interior rows take 6 (M0 - 2) of them
    if (M0 >= 16 && cfg.threads <= 256) return launch_tma_inst<TX, M0, kCluster, 256, 1>(cfg, tm, prm, st);
    if (cfg.threads <= 256) return launch_tma_inst<TX, M0, kCluster, 256, 2>(cfg, tm, prm, st);
    if (cfg.threads <= 512) return launch_tma_inst<TX, M0, kCluster, 512, 1>(cfg, tm, prm, st);
    return launch_tma_inst<TX, M0, kCluster, 1024, 1>(cfg, tm, prm, st);
}

template <int TX, bool kCluster>
inline cudaError_t launch_tma_tx(TmaFusedConfig &cfg, const CUtensorMap *tm, const TmaFusedParams &prm,
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

// a, b, c, d: batch base pointers (slice 0 of the launch), 16-byte aligned; x: 8-byte aligned.
inline cudaError_t launch_tma_fused(TmaFusedConfig &cfg, const double *a, const double *b,
                                    const double *c, const double *d, double *x, int nx, int ny,
                                    int nzs, long long rs, long long os, bool axis_z, bool periodic,
                                    cudaStream_t st)
{
    CUtensorMap tm[5];
    const void *ptr[5] = {a, b, c, d, x};
    for (int i = 0; i < 5 && nzs > 0; ++i) {
        if (i == 4 && !cfg.xaxis) { tm[4] = tm[3]; break; }      // x is stored from registers
        if (cfg.xaxis ? !make_xsweep_tensor_map(&tm[i], ptr[i], ny, nx, nzs, cfg.lines)
                      : !make_slab_tensor_map(&tm[i], ptr[i], nx, ny, nzs, rs, os, axis_z, cfg.lines, cfg.box_rows))
            return cudaErrorInvalidValue;
    }
    TmaFusedParams prm;
    prm.nx = nx; prm.ny = ny; prm.nzs = nzs;
    prm.x = x;
    prm.rs = rs; prm.os = os; prm.axis_z = axis_z ? 1 : 0; prm.periodic = periodic ? 1 : 0;
    prm.CL = cfg.cluster; prm.R = cfg.rows; prm.W = cfg.leaves;
    prm.xtiles = (nx + cfg.lines - 1) / cfg.lines;
    prm.ntiles = prm.xtiles * nzs;
    prm.box_rows = cfg.box_rows; prm.nbox = cfg.rows / cfg.box_rows;
    const bool cl = cfg.cluster > 1;
    if (cfg.xaxis)
        return cl ? launch_tma_inst<16, 16, true, 256, 1, true>(cfg, tm, prm, st)
                  : launch_tma_inst<16, 16, false, 256, 1, true>(cfg, tm, prm, st);
    switch (cfg.lines) {
    case 32: return cl ? launch_tma_tx<32, true>(cfg, tm, prm, st) : launch_tma_tx<32, false>(cfg, tm, prm, st);
    case 16: return cl ? launch_tma_tx<16, true>(cfg, tm, prm, st) : launch_tma_tx<16, false>(cfg, tm, prm, st);
    case 8: return cl ? launch_tma_tx<8, true>(cfg, tm, prm, st) : launch_tma_tx<8, false>(cfg, tm, prm, st);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace tdma
