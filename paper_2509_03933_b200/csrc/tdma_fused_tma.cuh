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
    int threads = 0;    // W * TX (the launch adds idle lanes up to a whole warp)
    int box_rows = 0;   // rows per TMA box (<= 256), divides R
    int slots = 0;      // NA: ring slots of one raw array each (4 = single-buffered tile ... 8 = two tiles)
    int max_clusters = 0;  // co-resident clusters (persistent grid size), filled at first launch
    bool xaxis = false;    // x sweep: 16-row leaves, swizzled boxes, staging tile for x
    size_t smem = 0;
    // the tensor maps of the last launches, keyed by the five base pointers and the slice count: plain
    // stream launches (no CUDA graph) of the same slab do not encode 5 maps per launch again
    struct MapSet { const void *ptr[5]; int nzs; CUtensorMap tm[5]; };
    static constexpr int kMapSets = 16;
    MapSet maps[kMapSets];
    int nmaps = 0, next_map = 0;
};

struct TmaFusedParams {
    double *x;          // batch base of the output
    long long rs, os;   // element stride between rows of a line / between slices of the caller's
                        // arrays (y sweep: nx, nx*ny; z sweep: nx*ny, nx)
    int axis_z;         // 0: rows = tensor dim 1, slices = dim 2;  1: rows = dim 2, slices = dim 1
    int periodic;       // cyclic lines: x_{-1} = x_{n-1}, x_n = x_0 (a_0, c_{n-1} are used)
    int nx, ny, nzs;    // ny = rows per line, nzs = slices in this launch
    int CL, R, W, NS;
    int xtiles, ntiles;
    int box_rows, nbox;
    // STAGED variant (kStage 1 / 2, tdma_staged.cu): reduced system of the batch in HBM, [2 Pe][Lb]
    // doubles, line fastest, unit diagonal; lp = tree levels run inside the CTA (the nodes of that
    // level are the partitions whose boundary equations are exchanged), lp_shift = log2(leaves per node)
    int pair = 0;       // 1: a cluster takes two ADJACENT x tiles one after the other (64-byte row segments:
                        // the pair shares 128-byte lines, fetched whole by the first tile's copies)
    double *red_a = nullptr, *red_c = nullptr, *red_d = nullptr;
    const double *red_y = nullptr;
    long long Lb = 0;
    int lp = 0, lp_shift = 0;
    // y-slab decomposition (tdma_slab.cu): this launch holds rows row0 .. row0 + ny - 1 of lines of
    // ny_total rows (0: the launch holds whole lines); Ls > 0: the reduced rows go to / the boundary
    // unknowns come from the all-to-all buffers send[dest][Pl][6][Ls] (red_a) / yrecv[src][2 Pl][Ls]
    // (red_y), dest = src = line / Ls, Pl = exchanged partitions of this rank
    int row0 = 0, ny_total = 0, Pl = 0;
    long long Ls = 0;
    // peer stores (tdma_slab_stage_a_peer): block `dest` of the send buffer is written straight into
    // rank dest's receive buffer, red_peer[dest] + red_peer_off (device table of nranks pointers)
    double *const *red_peer = nullptr;
    long long red_peer_off = 0;
};

// Dynamic shared memory of one CTA: NA ring slots of one raw array [R][TX] each, the x staging
// tile [R][TX], node buffer (2 planes of [2W][TX] 16-byte pairs), two inboxes of the
// cluster-level system (2 planes of [2 CL][TX] pairs each), NA + 2 mbarriers.
__host__ __device__ inline size_t tma_fused_smem_bytes(int TX, int R, int W, int CL, int NA, bool xaxis = false)
{
    (void)xaxis;
    const size_t raw = ((size_t)NA + 1) * R * TX * sizeof(double);
    const size_t node = (size_t)2 * 2 * W * TX * 16;
    const size_t inbox = CL > 1 ? (size_t)2 * 2 * 2 * CL * TX * 16 : 0;
    return raw + node + inbox + 128;
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
__device__ __forceinline__ void tma_load_4d(void *dst, const CUtensorMap *tm, int c0, int c1, int c2, int c3, uint64_t *bar)
{
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
        ::"r"(smem_u32(dst)), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tma_store_4d(const CUtensorMap *tm, int c0, int c1, int c2, int c3, const void *src)
{
    asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.bulk_group [%0, {%1, %2, %3, %4}], [%5];"
                 ::"l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(src)) : "memory");
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
// The lanes of a warp work on consecutive lines of the same row: conflict-free.  A row the tree
// eliminated keeps (a, c) in its AB slot and d (later x) in the D half of its CD slot.
// NC = 2 (two right-hand sides of the same matrix: the re / im parts of a complex field,
// tdma_shared_tma.cuh) adds a third plane of 8-byte entries, D1[row][line] at `d1`.
struct NodeBuf { uint32_t ab, plane, d1; };

template <int TX>
__device__ __forceinline__ uint32_t nb_ab(const NodeBuf &nb, int row, int lx) { return nb.ab + (uint32_t)(row * TX + lx) * 16u; }

// address of the D1 entry that belongs to the AB slot at address o
__device__ __forceinline__ uint32_t nb_d1(const NodeBuf &nb, uint32_t o) { return nb.d1 + ((o - nb.ab) >> 1); }

// the right-hand side(s) of the row whose AB slot is at o: cd = its CD pair, already loaded
template <int NC>
__device__ __forceinline__ void nb_load_d(const NodeBuf &nb, uint32_t o, const double2 &cd, double (&d)[NC])
{
    d[0] = cd.y;
    if (NC == 2) d[NC - 1] = lds1(nb_d1(nb, o));
}
template <int NC>
__device__ __forceinline__ void nb_store_d(const NodeBuf &nb, uint32_t o, const double (&d)[NC])
{
    sts1(o + nb.plane + 8, d[0]);
    if (NC == 2) sts1(nb_d1(nb, o), d[NC - 1]);
}
template <int NC>
__device__ __forceinline__ void nb_load_donly(const NodeBuf &nb, uint32_t o, double (&d)[NC])
{
    d[0] = lds1(o + nb.plane + 8);
    if (NC == 2) d[NC - 1] = lds1(nb_d1(nb, o));
}

// ------------------------------------------------------------------------------------------
// K-ary merge of boundary equations (the levels above the leaves, and the cluster-level system
// of cyclic lines).
//
// K consecutive nodes of S rows each (first equation in the node's first row, last equation in
// its last row) form a 2K-row tridiagonal system in u_0 = x_first(node 0), u_1 = x_last(node 0),
// u_2 = x_first(node 1), ..., u_{2K-1} = x_last(node K-1):
//     row i:  s_i u_{i-1} + b_i u_i + c_i u_{i+1} = d_i        (u_{-1} = x_prev, u_{2K} = x_next).
// The merged node's two equations come from two INDEPENDENT sweeps, run by two threads, carried
// un-normalised (no division on the serial chain) and rescaled by exact powers of two:
//   kmerge_fwd, rows 1 .. 2K-1, u_0 kept as a parameter:  al u_0 + be u_i + ga u_{i+1} = de,
//       al_i = -s_i al_{i-1},  be_i = be_{i-1} b_i - s_i ga_{i-1},  ga_i = be_{i-1} c_i,
//       de_i = be_{i-1} d_i - s_i de_{i-1};   row 2K-1 couples (u_0, u_{2K-1}, x_next): the merged
//       LAST equation, written to the group's last row;
//   kmerge_bwd, rows 2K-2 .. 0, u_{2K-1} kept as a parameter:  al u_{i-1} + be u_i + ga u_{2K-1} = de,
//       al_i = be_{i+1} s_i,  be_i = be_{i+1} b_i - c_i al_{i+1},  ga_i = -c_i ga_{i+1},
//       de_i = be_{i+1} d_i - c_i de_{i+1};   row 0 couples (x_prev, u_0, u_{2K-1}): the merged
//       FIRST equation, written to the group's first row.
// Neither sweep writes a row the other one reads.  The interior rows 1 .. 2K-2 stay untouched
// until kmerge_tails (a third thread, off the serial chain) turns them into
//     u_i = d_i - a_i u_0 - c_i u_{2K-1}.                                   K = 0: runtime k.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ int krow(int g, int k, int S, int i) { return (g * k + (i >> 1)) * S + ((i & 1) ? S - 1 : 0); }

template <int TX, int K, int NC = 1>
__device__ __forceinline__ void kmerge_fwd(const NodeBuf &nb, int lx, int g, int S, int kk)
{
    const int k = K > 0 ? K : kk;
    uint32_t o = nb_ab<TX>(nb, krow(g, k, S, 1), lx);
    double2 ab = lds2(o), cd = lds2(o + nb.plane);
    double al = ab.x, be = ab.y, ga = cd.x, de[NC], dn[NC];
    nb_load_d<NC>(nb, o, cd, de);
    o = nb_ab<TX>(nb, krow(g, k, S, 2), lx);
    ab = lds2(o); cd = lds2(o + nb.plane); nb_load_d<NC>(nb, o, cd, dn);
#pragma unroll
    for (int i = 2; i < 2 * k; ++i) {
        const double s = ab.x, b = ab.y, c = cd.x;
        double d[NC];
#pragma unroll
        for (int q = 0; q < NC; ++q) d[q] = dn[q];
        if (i + 1 < 2 * k) {                                  // next row's loads go out first
            o = nb_ab<TX>(nb, krow(g, k, S, i + 1), lx);
            ab = lds2(o); cd = lds2(o + nb.plane); nb_load_d<NC>(nb, o, cd, dn);
        }
        const double nbe = fma(be, b, -(s * ga));
#pragma unroll
        for (int q = 0; q < NC; ++q) de[q] = fma(be, d[q], -(s * de[q]));
        al = -(s * al); ga = be * c; be = nbe;
        if (i == 2 * k - 1 || ((i - 1) & 7) == 0) {          // rescale: last step, and every 8th of a long sweep
            const double sc = pow2_unscale(be);
#pragma unroll
            for (int q = 0; q < NC; ++q) de[q] *= sc;
            al *= sc; ga *= sc; be *= sc;
        }
    }
    sts2(o, al, be); sts2(o + nb.plane, ga, de[0]);           // o: the group's last row
    if (NC == 2) sts1(nb_d1(nb, o), de[NC - 1]);
}

template <int TX, int K, int NC = 1>
__device__ __forceinline__ void kmerge_bwd(const NodeBuf &nb, int lx, int g, int S, int kk)
{
    const int k = K > 0 ? K : kk;
    uint32_t o = nb_ab<TX>(nb, krow(g, k, S, 2 * k - 2), lx);
    double2 ab = lds2(o), cd = lds2(o + nb.plane);
    double al = ab.x, be = ab.y, ga = cd.x, de[NC], dn[NC];
    nb_load_d<NC>(nb, o, cd, de);
    o = nb_ab<TX>(nb, krow(g, k, S, 2 * k - 3), lx);
    ab = lds2(o); cd = lds2(o + nb.plane); nb_load_d<NC>(nb, o, cd, dn);
#pragma unroll
    for (int i = 2 * k - 3; i >= 0; --i) {
        const double s = ab.x, b = ab.y, c = cd.x;
        double d[NC];
#pragma unroll
        for (int q = 0; q < NC; ++q) d[q] = dn[q];
        if (i > 0) {
            o = nb_ab<TX>(nb, krow(g, k, S, i - 1), lx);
            ab = lds2(o); cd = lds2(o + nb.plane); nb_load_d<NC>(nb, o, cd, dn);
        }
        const double nbe = fma(be, b, -(c * al));
#pragma unroll
        for (int q = 0; q < NC; ++q) de[q] = fma(be, d[q], -(c * de[q]));
        ga = -(c * ga); al = be * s; be = nbe;
        if (i == 0 || ((2 * k - 2 - i) & 7) == 0) {
            const double sc = pow2_unscale(be);
#pragma unroll
            for (int q = 0; q < NC; ++q) de[q] *= sc;
            al *= sc; ga *= sc; be *= sc;
        }
    }
    sts2(o, al, be); sts2(o + nb.plane, ga, de[0]);           // o: the group's first row
    if (NC == 2) sts1(nb_d1(nb, o), de[NC - 1]);
}

// Interior rows i = 1 .. 2K-2 of a group, from their ORIGINAL equations (the merge sweeps only
// read them): modified Thomas forward sweep with u_0 as a parameter (normalised; this runs off
// the serial chain), then the backward sweep into
//     u_i = d_i - a_i u_0 - c_i u_{2K-1} :   AB slot <- (a, c),  D <- d.
template <int TX, int K, int NC = 1>
__device__ __forceinline__ void kmerge_tails(const NodeBuf &nb, int lx, int g, int S, int kk)
{
    const int k = K > 0 ? K : kk;
    double a = 0.0, c = 0.0, d[NC];
#pragma unroll
    for (int q = 0; q < NC; ++q) d[q] = 0.0;
    for (int i = 1; i <= 2 * k - 2; ++i) {
        const uint32_t o = nb_ab<TX>(nb, krow(g, k, S, i), lx);
        const double2 ab = lds2(o), cd = lds2(o + nb.plane);
        double di[NC];
        nb_load_d<NC>(nb, o, cd, di);
        if (i == 1) {
            const double inv = rcp_nr(ab.y);
            a = ab.x * inv; c = cd.x * inv;
#pragma unroll
            for (int q = 0; q < NC; ++q) d[q] = di[q] * inv;
        } else {
            const double inv = rcp_nr(fma(-ab.x, c, ab.y));
#pragma unroll
            for (int q = 0; q < NC; ++q) d[q] = fma(-ab.x, d[q], di[q]) * inv;
            a = -(ab.x * a) * inv;
            c = cd.x * inv;
        }
        sts2(o, a, c); nb_store_d<NC>(nb, o, d);
    }
    // a, c, d: row 2K-2, already in final form
    for (int i = 2 * k - 3; i >= 1; --i) {
        const uint32_t o = nb_ab<TX>(nb, krow(g, k, S, i), lx);
        const double2 ac = lds2(o);
        double di[NC];
        nb_load_donly<NC>(nb, o, di);
#pragma unroll
        for (int q = 0; q < NC; ++q) d[q] = fma(-ac.y, d[q], di[q]);
        a = fma(-ac.y, a, ac.x);
        c = -(ac.y * c);
        sts2(o, a, c); nb_store_d<NC>(nb, o, d);
    }
}

// The same in two steps for a HELPER thread that runs concurrently with the merge sweeps of the
// same level: kmerge_tails_regs reads the 2K-2 interior rows and leaves (a, c, d) in registers,
// kmerge_tails_store writes them back once the sweeps no longer read the rows.
template <int TX, int K, int NC = 1>
__device__ __forceinline__ void kmerge_tails_regs(const NodeBuf &nb, int lx, int g, int S, double (&a)[6], double (&c)[6],
                                                  double (&d)[6][NC])
{
    constexpr int NI = 2 * K - 2;
    double2 ab[NI], cd[NI];
#pragma unroll
    for (int j = 0; j < NI; ++j) {
        const uint32_t o = nb_ab<TX>(nb, krow(g, K, S, j + 1), lx);
        ab[j] = lds2(o); cd[j] = lds2(o + nb.plane);
        nb_load_d<NC>(nb, o, cd[j], d[j]);
    }
    double inv = rcp_nr(ab[0].y);
    a[0] = ab[0].x * inv; c[0] = cd[0].x * inv;
#pragma unroll
    for (int q = 0; q < NC; ++q) d[0][q] *= inv;
#pragma unroll
    for (int j = 1; j < NI; ++j) {
        inv = rcp_nr(fma(-ab[j].x, c[j - 1], ab[j].y));
#pragma unroll
        for (int q = 0; q < NC; ++q) d[j][q] = fma(-ab[j].x, d[j - 1][q], d[j][q]) * inv;
        a[j] = -(ab[j].x * a[j - 1]) * inv;
        c[j] = cd[j].x * inv;
    }
#pragma unroll
    for (int j = NI - 2; j >= 0; --j) {
#pragma unroll
        for (int q = 0; q < NC; ++q) d[j][q] = fma(-c[j], d[j + 1][q], d[j][q]);
        a[j] = fma(-c[j], a[j + 1], a[j]);
        c[j] = -(c[j] * c[j + 1]);
    }
}

template <int TX, int K, int NC = 1>
__device__ __forceinline__ void kmerge_tails_store(const NodeBuf &nb, int lx, int g, int S, const double (&a)[6],
                                                   const double (&c)[6], const double (&d)[6][NC])
{
#pragma unroll
    for (int j = 0; j < 2 * K - 2; ++j) {
        const uint32_t o = nb_ab<TX>(nb, krow(g, K, S, j + 1), lx);
        sts2(o, a[j], c[j]); nb_store_d<NC>(nb, o, d[j]);
    }
}

// u_i of a group (i = 0 .. 2k-1) from the group's x_first / x_last.
template <int TX, int NC = 1>
__device__ __forceinline__ void kmerge_value_n(const NodeBuf &nb, int lx, int g, int S, int k, int i,
                                               const double (&xf)[NC], const double (&xl)[NC], double (&out)[NC])
{
#pragma unroll
    for (int q = 0; q < NC; ++q) out[q] = i == 0 ? xf[q] : xl[q];
    if (i == 0 || i == 2 * k - 1) return;
    const uint32_t o = nb_ab<TX>(nb, krow(g, k, S, i), lx);
    const double2 ac = lds2(o);
    double di[NC];
    nb_load_donly<NC>(nb, o, di);
#pragma unroll
    for (int q = 0; q < NC; ++q) out[q] = fma(-ac.y, xl[q], fma(-ac.x, xf[q], di[q]));
}
template <int TX>
__device__ __forceinline__ double kmerge_value(const NodeBuf &nb, int lx, int g, int S, int k, int i, double xf, double xl)
{
    if (i == 0) return xf;
    if (i == 2 * k - 1) return xl;
    const uint32_t o = nb_ab<TX>(nb, krow(g, k, S, i), lx);
    const double2 ac = lds2(o);
    return fma(-ac.y, xl, fma(-ac.x, xf, lds1(o + nb.plane + 8)));
}

// Cluster-level system of a PLAIN (non-cyclic) line, rows i = 0 .. n-1 of `tb` (s_0 = c_{n-1} = 0):
// the CTA needs only its own two unknowns u_p, u_{p+1} (p = 2 * rank), so it eliminates towards
// them from both ends, un-normalised (no division on the chain),
//     forward   be u_i + ga u_{i+1} = de ,  i = 0 .. p      (be_i = be_{i-1} b_i - s_i ga_{i-1}, ...)
//     backward  al u_{i-1} + bb u_i = dd ,  i = n-1 .. p+1  (bb_i = bb_{i+1} b_i - c_i al_{i+1}, ...)
// and solves the remaining 2 x 2 system.  The two sweeps are independent chains of p and n-2-p
// steps that run interleaved in one thread; one reciprocal in total.
template <int TX, int NC = 1>
__device__ __forceinline__ void cluster_solve_two_sided(const NodeBuf &tb, int lx, int n, int p, double (&up)[NC], double (&up1)[NC])
{
    uint32_t of = nb_ab<TX>(tb, 0, lx), ob = nb_ab<TX>(tb, n - 1, lx);
    const uint32_t step = TX * 16u;
    double2 t0 = lds2(of), t1 = lds2(of + tb.plane), t2 = lds2(ob), t3 = lds2(ob + tb.plane);
    double be = t0.y, ga = t1.x, de[NC];                // row 0
    double al = t2.x, bb = t2.y, dd[NC];                // row n-1
    nb_load_d<NC>(tb, of, t1, de);
    nb_load_d<NC>(tb, ob, t3, dd);
    const int nf = p, nbk = n - 2 - p;
    const int nmax = nf > nbk ? nf : nbk;
    double2 fab = make_double2(0.0, 1.0), fcd = make_double2(0.0, 0.0), bab = fab, bcd = fcd;
    double fdn[NC], bdn[NC];
#pragma unroll
    for (int q = 0; q < NC; ++q) fdn[q] = bdn[q] = 0.0;
    if (nf > 0) { of += step; fab = lds2(of); fcd = lds2(of + tb.plane); nb_load_d<NC>(tb, of, fcd, fdn); }
    if (nbk > 0) { ob -= step; bab = lds2(ob); bcd = lds2(ob + tb.plane); nb_load_d<NC>(tb, ob, bcd, bdn); }
    for (int j = 0; j < nmax; ++j) {
        const double fs = fab.x, fb_ = fab.y, fc_ = fcd.x;
        const double bs = bab.x, bb_ = bab.y, bc_ = bcd.x;
        double fd_[NC], bd_[NC];
#pragma unroll
        for (int q = 0; q < NC; ++q) { fd_[q] = fdn[q]; bd_[q] = bdn[q]; }
        const bool fw = j < nf, bw = j < nbk;
        if (j + 1 < nf) { of += step; fab = lds2(of); fcd = lds2(of + tb.plane); nb_load_d<NC>(tb, of, fcd, fdn); }
        if (j + 1 < nbk) { ob -= step; bab = lds2(ob); bcd = lds2(ob + tb.plane); nb_load_d<NC>(tb, ob, bcd, bdn); }
        const bool rs = (j & 7) == 7;                          // rescale every 8th step of a long sweep
        if (fw) {
            const double nbe = fma(be, fb_, -(fs * ga));
#pragma unroll
            for (int q = 0; q < NC; ++q) de[q] = fma(be, fd_[q], -(fs * de[q]));
            ga = be * fc_; be = nbe;
            if (rs) {
                const double sc = pow2_unscale(be);
#pragma unroll
                for (int q = 0; q < NC; ++q) de[q] *= sc;
                ga *= sc; be *= sc;
            }
        }
        if (bw) {
            const double nbb = fma(bb, bb_, -(bc_ * al));
#pragma unroll
            for (int q = 0; q < NC; ++q) dd[q] = fma(bb, bd_[q], -(bc_ * dd[q]));
            al = bb * bs; bb = nbb;
            if (rs) {
                const double sc = pow2_unscale(bb);
#pragma unroll
                for (int q = 0; q < NC; ++q) dd[q] *= sc;
                al *= sc; bb *= sc;
            }
        }
    }
    const double inv = rcp_nr(fma(be, bb, -(ga * al)));
#pragma unroll
    for (int q = 0; q < NC; ++q) {
        up[q] = fma(de[q], bb, -(ga * dd[q])) * inv;
        up1[q] = fma(be, dd[q], -(al * de[q])) * inv;
    }
}

// Root of a tree: first equation  A x_prev + B x_f + C x_l = D  (row 0), last equation
// A x_f + B x_l + C x_next = D  (row rl)  ->  x_f, x_l into D.  Plain lines: the root's A_first and
// C_last are 0.  Cyclic lines (wrap): x_prev = x_l and x_next = x_f, i.e. the periodic coupling is
// resolved here, at the top of the recursion, as  B_f x_f + (A_f + C_f) x_l = D_f ,
// (A_l + C_l) x_f + B_l x_l = D_l  -- no Sherman-Morrison correction is needed.
template <int TX, int NC = 1>
__device__ __forceinline__ void solve_root(const NodeBuf &nb, int lx, int rl, bool wrap)
{
    const uint32_t oF = nb_ab<TX>(nb, 0, lx), oL = nb_ab<TX>(nb, rl, lx);
    const double2 abf = lds2(oF), cdf = lds2(oF + nb.plane), abl = lds2(oL), cdl = lds2(oL + nb.plane);
    double df[NC], dl[NC], xf[NC], xl[NC];
    nb_load_d<NC>(nb, oF, cdf, df);
    nb_load_d<NC>(nb, oL, cdl, dl);
    const double Cf = wrap ? cdf.x + abf.x : cdf.x, Al = wrap ? abl.x + cdl.x : abl.x;
    const double inv = rcp_nr(fma(abf.y, abl.y, -(Cf * Al)));
#pragma unroll
    for (int q = 0; q < NC; ++q) {
        xl[q] = fma(abf.y, dl[q], -(Al * df[q])) * inv;
        xf[q] = fma(abl.y, df[q], -(Cf * dl[q])) * inv;
    }
    nb_store_d<NC>(nb, oL, xl);
    nb_store_d<NC>(nb, oF, xf);
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

// Back-substitution of the leaf from registers given its first and last unknown: row j of the
// leaf goes to the x staging tile at sx + j * row_bytes (shared-space address).
template <int M0>
__device__ __forceinline__ void leaf_back(const LeafRegs<M0> &R, double xf, double xl, uint32_t sx, uint32_t row_bytes)
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
        sts1(sx + (uint32_t)(h * H) * row_bytes, first[h]);
        sts1(sx + (uint32_t)(h * H + H - 1) * row_bytes, last[h]);
    }
#pragma unroll
    for (int r = H - 2; r >= 1; --r) {
#pragma unroll
        for (int h = 0; h < K; ++h) {
            xn[h] = fma(-R.ic[h][r - 1], xn[h], fma(-R.ia[h][r - 1], first[h], R.id[h][r - 1]));
            sts1(sx + (uint32_t)(h * H + r) * row_bytes, xn[h]);
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

// Named barrier over the tree threads (whole warps; a single warp needs __syncwarp only).
__device__ __forceinline__ void tree_sync(int nthreads, unsigned warp_mask)
{
    if (nthreads > 32) asm volatile("bar.sync 1, %0;" ::"r"(nthreads) : "memory");
    else __syncwarp(warp_mask);
}
__device__ __forceinline__ void named_arrive(int id, int nthreads)
{
    asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
__device__ __forceinline__ void named_sync(int id, int nthreads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// kX: x sweep (lanes = TX lines along y, rows = x; M0 = 16 only).
//
// Threads: leaf = t / TX, lx = t % TX (a warp covers whole row segments, so tile reads,
// node-buffer accesses and x stores are coalesced / conflict-free); blockDim = W*TX rounded up to
// whole warps.
// Raw tile ring.  The four arrays of a tile are fetched one TMA copy group each, in the order
// the sweep needs them (b, a, c, d), into a ring of NA >= 4 array slots (array j of the cluster's
// q-th tile: n = 4q + j -> slot n % NA), each with its own mbarrier.  As soon as the sweep of tile
// q has consumed its four slots, arrays 4q+NA .. 4q+NA+3 are issued: with NA > 4, NA - 4 arrays
// of the next tile are in flight while a tile is being swept, so HBM never idles behind the
// sweep.  A TMA copy costs its issuing thread 150-200 cycles (measured), so the copies are
// issued by the LAST warp, which has no part in the tree that follows the sweep.
// x leaves the SM the same way: back-substitution writes the staging tile in shared memory and
// the last warp hands it to the TMA engine (one tensor store per box) after the NEXT tile's
// sweep -- an SM retires plain global stores at about a sector per cycle, which would block the
// load/store unit the sweep reads the raw tile with for > 1000 cycles per tile.
// kStage (STAGED variant: the paper's three stages as separate kernels with the
// partition segments staged on chip, nothing spilled):
//   0  the fused solve described above;
//   1  stage A: sweep + tree up to the partition level, the partitions' boundary equations
//      (unit diagonal) go to the reduced buffers in HBM; no back-substitution, x untouched;
//   2  stage C: the tile is fetched and reduced AGAIN (a', c', d' never leave the chip), the
//      partitions' boundary unknowns come from the reduced solution Y, then walk-down and leaf
//      back-substitution as in the fused solve.
//   kStage != 0: CTAs are independent (no cluster, no DSMEM): CL consecutive CTAs share a line tile.
template <int TX, int M0, bool kCluster, int MAXT, bool kX, int kStage = 0>
__global__ void __launch_bounds__(MAXT, 1)
fused_tma_kernel(const __grid_constant__ CUtensorMap tm_a, const __grid_constant__ CUtensorMap tm_b,
                 const __grid_constant__ CUtensorMap tm_c, const __grid_constant__ CUtensorMap tm_d,
                 const __grid_constant__ CUtensorMap tm_x, const TmaFusedParams prm)
{
    static_assert(!kX || M0 == 16, "x sweeps use 16-row (128-byte) leaves");
    static_assert(kStage == 0 || (!kCluster && !kX), "staged kernels: independent CTAs, y / z sweeps");
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    const int R = prm.R, CL = prm.CL, W = prm.W, NA = prm.NS;
    const int arr = R * TX;
    double *const raw = reinterpret_cast<double *>(smem_raw);         // NA slots of one array [R][TX]
    double *sX = raw + (size_t)NA * arr;                              // x staging tile
    double *node = sX + arr;
    NodeBuf nb;                                                       // node buffer, 2 planes of [2W][TX] pairs
    nb.ab = ptx::smem_u32(node); nb.plane = (uint32_t)(2 * W * TX) * 16u; nb.d1 = 0;
    const int NTR = 2 * CL;                                           // rows of the cluster-level system
    NodeBuf tb0;                                                      // inbox of parity 0: 2 planes of [NTR][TX]
    tb0.ab = nb.ab + 2u * nb.plane; tb0.plane = (uint32_t)(NTR * TX) * 16u; tb0.d1 = 0;
    const uint32_t inbox_bytes = kCluster ? 2u * tb0.plane : 0u;
    uint64_t *bar = reinterpret_cast<uint64_t *>(smem_raw + (tb0.ab + 2u * inbox_bytes - ptx::smem_u32(smem_raw)));
    // bar[0 .. NA-1]: slot full; bar[NA], bar[NA+1]: inboxes

    const int t = threadIdx.x;
    const int NT = W * TX;
    const bool act = t < NT;
    // tree threads: all warps but the last (which issues the copies); a single warp does both
    const int tree_threads = (int)blockDim.x > 32 ? (int)blockDim.x - 32 : NT;
    const bool tree = t < tree_threads && act;
    const int Wt = tree_threads / TX;
    const unsigned tmask = __ballot_sync(0xffffffffu, tree);
    unsigned crank = 0;
    if (kCluster) crank = cg::this_cluster().block_rank();
    if (kStage != 0) crank = blockIdx.x % CL;
    const int g = blockIdx.x / CL, NC = gridDim.x / CL;        // cluster index / number of clusters
    const int y0 = (int)crank * R;

    if (t == 0) {
        for (int i = 0; i < NA + 2; ++i) ptx::mbar_init(&bar[i], 1);
        ptx::fence_mbar_init();
    }
    __syncthreads();                    // mbarriers initialised before anyone uses them
    // split-phase cluster barrier: "every CTA of the cluster has started and initialised its
    // inbox mbarriers" must hold before the first remote store; the matching wait sits right
    // before the first exchange
    if (kCluster) asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");

    // TMA copies of one raw array, by the lanes of the last warp
    const int issue_lane = t - ((int)blockDim.x - 32 > 0 ? (int)blockDim.x - 32 : 0);   // >= 0: issuing warp
    const uint32_t arr_bytes = (uint32_t)(arr * sizeof(double));
    // the cluster's q-th tile
    auto tile_of = [&](int q) { return prm.pair ? (((q >> 1) * NC + g) << 1) + (q & 1) : g + q * NC; };
    auto issue_array = [&](int n) {
        const int tile = tile_of(n >> 2), j = n & 3;
        if (tile >= prm.ntiles) return;
        const int s = n % NA;
        const int x0 = (tile % prm.xtiles) * TX, k = tile / prm.xtiles;
        double *const dst = raw + (size_t)s * arr;
        const CUtensorMap *const tm = j == 0 ? &tm_b : (j == 1 ? &tm_a : (j == 2 ? &tm_c : &tm_d));
        if (issue_lane == 0) ptx::mbar_expect_tx(&bar[s], arr_bytes);
        if (kX) {
            // x sweep: the line axis is viewed as (16 x, leaf) -- tensor (16, lanes, nrows / 16, slices)
            // -- so ONE copy of box (16, TX, W, 1) brings the CTA's W leaves of all TX lines, laid out
            // [leaf][line][16 x] with the 128-byte swizzle keyed by the line; x0 = first line
            if (issue_lane == 0) ptx::tma_load_4d(dst, tm, 0, x0, y0 >> 4, k, &bar[s]);
        } else if (issue_lane == 0) {
            for (int q = 0; q < prm.nbox; ++q) {
                const int yy = y0 + q * prm.box_rows;
                ptx::tma_load_3d(dst + q * prm.box_rows * TX, tm, x0, prm.axis_z ? k : yy, prm.axis_z ? yy : k, &bar[s]);
            }
        }
    };
    // the staging tile of tile `tile` -> x (TMA clips the ragged last x tile)
    auto store_x = [&](int tile) {
        const int x0 = (tile % prm.xtiles) * TX, k = tile / prm.xtiles;
        if (kX) {
            if (issue_lane == 0) ptx::tma_store_4d(&tm_x, 0, x0, y0 >> 4, k, sX);
        } else if (issue_lane == 0) {
            for (int q = 0; q < prm.nbox; ++q) {
                const int yy = y0 + q * prm.box_rows;
                ptx::tma_store_3d(&tm_x, x0, prm.axis_z ? k : yy, prm.axis_z ? yy : k, sX + q * prm.box_rows * TX);
            }
        }
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    };
    if (issue_lane >= 0) for (int n = 0; n < NA; ++n) issue_array(n);

    const int lx = t % TX, leaf = t / TX;
    const int ny_line = (kStage != 0 && prm.ny_total > 0) ? prm.ny_total : prm.ny;      // rows of the whole line
    const int row_g = (kStage != 0 ? prm.row0 : 0) + y0 + leaf * M0;                     // global row of the leaf
    const bool first_leaf = !prm.periodic && row_g == 0;
    const bool last_leaf = !prm.periodic && row_g + M0 == ny_line;
    const int o0 = leaf * M0 * TX + lx;
    // levels above the leaves: 4-ary merges (2-ary when the node count is not a multiple of 4)
    // level l merges k = 2^lkb nodes of S = 2 << cum rows (cum = sum of the lkb below); packed into
    // two words (a local array indexed by the level would live in local memory)
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

    // Static split of the tree threads, by whole warps:
    //   CRITICAL warps [0, cw): their thread rows run the merge sweeps of every level, synchronise
    //     among themselves only (named barrier 1), send the CTA's node and solve the cluster-level
    //     system -- the serial chain of a tile;
    //   HELPER warps [cw, tree warps): their thread rows compute the interior-row forms
    //     (kmerge_tails) of every level CONCURRENTLY with that level's merge sweeps, in registers,
    //     and store them once the sweeps have signalled (bar.arrive on named barrier 2 + level,
    //     which costs the critical warps nothing) that they no longer read the rows.
    // Without helper warps (small tiles) the critical rows do the interior rows themselves.
    const int G0 = nl > 0 ? level_groups(0) : 0;
    const int rpw = TX >= 32 ? 1 : 32 / TX;                           // thread rows per warp
    const int crit_rows = Wt >= 2 * G0 ? 2 * G0 : (Wt >= G0 ? G0 : Wt);
    const int cw = (crit_rows + rpw - 1) / rpw;
    const bool helper_mode = nl > 0 && (int)blockDim.x > 32 && cw * 32 < tree_threads;
    const int help0 = helper_mode ? cw * rpw : Wt;                   // first helper row
    const int nhelp = Wt - help0;
    const int mrows = helper_mode ? crit_rows : Wt;                  // rows that share the merges of a level
    const int crit_threads = helper_mode ? cw * 32 : tree_threads;
    const bool crit = tree && leaf < help0, helper = tree && !crit;
    int it = 0, sn = 0, pn = 0;
    for (int tile = tile_of(0); tile < prm.ntiles; tile = tile_of(++it)) {
        const int par = it & 1;
        NodeBuf tb = tb0;                                      // this tile's inbox
        tb.ab += (uint32_t)par * inbox_bytes;
        // arm this tile's inbox: 4 doubles per (node equation, line) from every CTA
        if (kCluster && t == 0) ptx::mbar_expect_tx(&bar[NA + par], (unsigned)(4 * NTR * TX * sizeof(double)));
        const int n0 = 4 * it;
        // ring slot / mbarrier phase of the tile's four arrays, advanced without divisions:
        // (sn, pn) = (n0 % NA, (n0 / NA) & 1); array j sits j slots further (at most one wrap, NA >= 4)
        int sl[4], ph[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            sl[j] = sn + j; ph[j] = pn;
            if (sl[j] >= NA) { sl[j] -= NA; ph[j] ^= 1; }
        }
        sn += 4;
        if (sn >= NA) { sn -= NA; pn ^= 1; }
        const double *__restrict__ sB = raw + (size_t)sl[0] * arr, *__restrict__ sA = raw + (size_t)sl[1] * arr;
        const double *__restrict__ sC = raw + (size_t)sl[2] * arr, *__restrict__ sD = raw + (size_t)sl[3] * arr;
        // staged kernels: where this thread's partition sits in the reduced buffers; stage C fetches its
        // two boundary unknowns now, a whole sweep ahead of their use
        long long red_l = -1;
        double y_first = 0.0, y_last = 0.0;
        if (kStage != 0) {
            const int xt_ = tile % prm.xtiles, k_ = tile / prm.xtiles;
            if (xt_ * TX + lx < prm.nx) red_l = (long long)k_ * prm.nx + xt_ * TX + lx;
            if (kStage == 2 && act && red_l >= 0) {
                const long long pg = (long long)crank * (W >> prm.lp_shift) + (leaf >> prm.lp_shift);
                if (prm.Ls > 0) {       // y-slab: yrecv[src][2 Pl][Ls]
                    const long long src = red_l / prm.Ls, j = red_l - src * prm.Ls;
                    const double *yp = prm.red_y + ((src * 2 * prm.Pl + 2 * pg) * prm.Ls + j);
                    y_first = __ldcg(yp); y_last = __ldcg(yp + prm.Ls);
                } else {
                    y_first = __ldcg(prm.red_y + 2 * pg * prm.Lb + red_l);
                    y_last = __ldcg(prm.red_y + (2 * pg + 1) * prm.Lb + red_l);
                }
            }
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) ptx::mbar_wait(&bar[sl[j]], (unsigned)ph[j]);

        // ---------------- leaves ----------------
        LeafRegs<M0> regs;
        if (act) {
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
        __syncthreads();                // raw slots consumed, leaf equations visible
        if (issue_lane >= 0) {
            for (int j = 0; j < 4; ++j) issue_array(n0 + NA + j);     // refill the four slots
            if (kStage != 1 && it > 0) store_x(tile_of(it - 1));       // x of the previous tile
        }
        if (kCluster && it == 0) asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");

        // ---------------- K-ary tree inside the CTA, bottom-up ----------------
        // The warp that issues the copies (the last one) takes no part in the tree, so the
        // 150-200 cycles per copy stay off the serial chain; everybody meets again before the
        // back-substitution.
        const int nlr = kStage != 0 ? prm.lp : nl;              // levels run inside the CTA
        if (helper && kStage != 1) {                            // stage A never walks down: no interior forms
            const int h = leaf - help0;
            int cum = 0;                                        // interior-row jobs of the levels below
            for (int l = 0; l < nlr; ++l) {
                const int k = level_k(l), S = level_S(l), groups = level_groups(l);
                int gq = (h - cum) % nhelp;
                if (gq < 0) gq += nhelp;
                double ta[6], tc[6], td[6][1];
                if (gq < groups) {
                    if (k == 4) kmerge_tails_regs<TX, 4>(nb, lx, gq, S, ta, tc, td);
                    else kmerge_tails_regs<TX, 2>(nb, lx, gq, S, ta, tc, td);
                }
                named_sync(2 + l, tree_threads);                // the merges of level l are done
                if (gq < groups) {
                    if (k == 4) kmerge_tails_store<TX, 4>(nb, lx, gq, S, ta, tc, td);
                    else kmerge_tails_store<TX, 2>(nb, lx, gq, S, ta, tc, td);
                    for (gq += nhelp; gq < groups; gq += nhelp) {   // more jobs than helper rows
                        if (k == 4) kmerge_tails<TX, 4>(nb, lx, gq, S, 4); else kmerge_tails<TX, 2>(nb, lx, gq, S, 2);
                    }
                }
                cum += groups;
            }
        }
        if (crit) {
            for (int l = 0; l < nlr; ++l) {
                const int k = level_k(l), S = level_S(l), groups = level_groups(l);
                for (int q = leaf; q < 2 * groups; q += mrows) {  // q < groups: forward, else backward sweep
                    if (q < groups) { if (k == 4) kmerge_fwd<TX, 4>(nb, lx, q, S, 4); else kmerge_fwd<TX, 2>(nb, lx, q, S, 2); }
                    else { if (k == 4) kmerge_bwd<TX, 4>(nb, lx, q - groups, S, 4); else kmerge_bwd<TX, 2>(nb, lx, q - groups, S, 2); }
                }
                if (helper_mode && kStage != 1) named_arrive(2 + l, tree_threads);
                tree_sync(crit_threads, tmask);
                if (!helper_mode && kStage != 1) {              // nobody reads the interior rows any more
                    for (int q = mrows - 1 - leaf; q < groups; q += mrows) {    // last rows first: row 0 goes on
                        if (k == 4) kmerge_tails<TX, 4>(nb, lx, q, S, 4); else kmerge_tails<TX, 2>(nb, lx, q, S, 2);
                    }
                }
            }

            // ---------------- cluster level ----------------
            // the CTA's node: first equation in node row 0, last equation in node row 2W-1
            if (kStage != 0) {
                // staged kernels: the exchange and the reduced solve are stage B's, through HBM
            } else if (!kCluster) {
                if (leaf == 0) solve_root<TX>(nb, lx, 2 * W - 1, prm.periodic != 0);
            } else {
                // A2B as an all-gather (the paper's MPI_Alltoall, with every rank
                // keeping a copy): asynchronous DSMEM stores that complete on the RECEIVER's mbarrier
                const uint32_t bar_s = ptx::smem_u32(&bar[NA + par]);
                for (int e = t; e < 4 * TX * CL; e += crit_threads) {
                    const int dest = e / (4 * TX), r = e - dest * 4 * TX;
                    const int piece = r / TX, l = r - piece * TX;  // piece: AB / CD of first, AB / CD of last
                    const int j = piece >> 1;
                    const uint32_t po = (piece & 1) ? 1u : 0u;
                    const double2 v = lds2(nb_ab<TX>(nb, j ? 2 * W - 1 : 0, l) + po * nb.plane);
                    const uint32_t dst = ptx::mapa(nb_ab<TX>(tb, (int)crank * 2 + j, l) + po * tb.plane, (unsigned)dest);
                    ptx::st_async_2f64(dst, v.x, v.y, ptx::mapa(bar_s, (unsigned)dest));
                }
                if (leaf == 0 && !prm.periodic) {
                    ptx::mbar_wait(&bar[NA + par], (unsigned)((it >> 1) & 1));
                    // Stage B: the 2 CL-row system; every CTA computes its own two unknowns (one
                    // thread per line), so no second exchange is needed (B2C is a local store)
                    double u0[1], u1[1];
                    cluster_solve_two_sided<TX>(tb, lx, NTR, 2 * (int)crank, u0, u1);
                    // into the CTA's own rows of its INBOX, not into the node rows: other warps of
                    // this CTA may still be reading those for their sends to the peers
                    sts1(nb_ab<TX>(tb, 2 * (int)crank, lx) + tb.plane + 8, u0[0]);
                    sts1(nb_ab<TX>(tb, 2 * (int)crank + 1, lx) + tb.plane + 8, u1[0]);
                } else if (leaf == 0) {
                    ptx::mbar_wait(&bar[NA + par], (unsigned)((it >> 1) & 1));
                    // cyclic lines: merge the CL nodes, resolve the wrap at the root, walk back
                    kmerge_fwd<TX, 0>(tb, lx, 0, 2, CL);
                    kmerge_bwd<TX, 0>(tb, lx, 0, 2, CL);
                    solve_root<TX>(tb, lx, NTR - 1, true);
                    kmerge_tails<TX, 0>(tb, lx, 0, 2, CL);
                    const double xf = lds1(nb_ab<TX>(tb, 0, lx) + tb.plane + 8), xl = lds1(nb_ab<TX>(tb, NTR - 1, lx) + tb.plane + 8);
                    const double v0 = kmerge_value<TX>(tb, lx, 0, 2, CL, 2 * (int)crank, xf, xl);
                    const double v1 = kmerge_value<TX>(tb, lx, 0, 2, CL, 2 * (int)crank + 1, xf, xl);
                    sts1(nb_ab<TX>(tb, 2 * (int)crank, lx) + tb.plane + 8, v0);
                    sts1(nb_ab<TX>(tb, 2 * (int)crank + 1, lx) + tb.plane + 8, v1);
                }
            }
        }
        // the TMA engine must have read the previous tile's x out of the staging tile
        if (issue_lane >= 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
        __syncthreads();
        if (kStage == 1) {
            // stage A's output: the two boundary equations of every partition (node of level lp),
            // normalised to unit diagonal, as rows 2 pg, 2 pg + 1 of the reduced system (the paper's
            // A2B gather, fused into the epilogue)
            const int Wp = W >> prm.lp_shift, S = 2 << prm.lp_shift;
            if (t < Wp * TX && red_l >= 0) {
                const long long pg = (long long)crank * Wp + leaf;      // leaf = t / TX: the node index here
                const uint32_t oF = nb_ab<TX>(nb, leaf * S, lx), oL = nb_ab<TX>(nb, leaf * S + S - 1, lx);
                const double2 abf = lds2(oF), cdf = lds2(oF + nb.plane), abl = lds2(oL), cdl = lds2(oL + nb.plane);
                const double invf = 1.0 / abf.y, invl = 1.0 / abl.y;
                if (prm.Ls > 0) {       // y-slab: send[dest][Pl][6][Ls] = (fa, fc, fd | pa, pc, pd)
                    const long long dest = red_l / prm.Ls, j = red_l - dest * prm.Ls;
                    double *sp = prm.red_peer ? prm.red_peer[dest] + (prm.red_peer_off + (long long)pg * 6 * prm.Ls + j)
                                              : prm.red_a + ((dest * prm.Pl + pg) * 6 * prm.Ls + j);
                    __stcg(sp, abf.x * invf); __stcg(sp + prm.Ls, cdf.x * invf); __stcg(sp + 2 * prm.Ls, cdf.y * invf);
                    __stcg(sp + 3 * prm.Ls, abl.x * invl); __stcg(sp + 4 * prm.Ls, cdl.x * invl); __stcg(sp + 5 * prm.Ls, cdl.y * invl);
                } else {
                    const long long q0 = 2 * pg * prm.Lb + red_l, q1 = q0 + prm.Lb;
                    __stcg(prm.red_a + q0, abf.x * invf); __stcg(prm.red_c + q0, cdf.x * invf); __stcg(prm.red_d + q0, cdf.y * invf);
                    __stcg(prm.red_a + q1, abl.x * invl); __stcg(prm.red_c + q1, cdl.x * invl); __stcg(prm.red_d + q1, cdl.y * invl);
                }
            }
            __syncthreads();            // the node rows are read before the next sweep rewrites them
            continue;
        }

        // ---------------- leaves: back-substitution from registers into the staging tile --------
        if (act) {
            // top-down through the tree in registers: every thread row walks from the CTA's node
            // to its own leaf (x_first / x_last of a child from those of its parent and the
            // interior-row form kmerge_tails left), no barrier, nothing written
            double xf, xl;                                      // cluster: stage B left them in the inbox
            if (kStage == 2) {
                xf = y_first; xl = y_last;                      // of this leaf's partition, from stage B's Y
            } else if (kCluster) {
                xf = lds1(nb_ab<TX>(tb, 2 * (int)crank, lx) + tb.plane + 8);
                xl = lds1(nb_ab<TX>(tb, 2 * (int)crank + 1, lx) + tb.plane + 8);
            } else {
                xf = lds1(nb_ab<TX>(nb, 0, lx) + nb.plane + 8);
                xl = lds1(nb_ab<TX>(nb, 2 * W - 1, lx) + nb.plane + 8);
            }
            for (int l = nlr - 1; l >= 0; --l) {
                const int k = level_k(l), S = level_S(l);
                const int node = leaf >> ((ccode >> (5 * l)) & 31u);        // my ancestor among this level's children
                const int gq = node >> ((kcode >> (2 * l)) & 3u), j = node & (k - 1);
                const double nf = kmerge_value<TX>(nb, lx, gq, S, k, 2 * j, xf, xl);
                const double nlast = kmerge_value<TX>(nb, lx, gq, S, k, 2 * j + 1, xf, xl);
                xf = nf; xl = nlast;
            }
            if constexpr (kX) leaf_back_x(regs, xf, xl, ptx::smem_u32(sX) + (uint32_t)(leaf * 16 * TX) * 8u, lx);
            else leaf_back<M0>(regs, xf, xl, ptx::smem_u32(sX) + (uint32_t)o0 * 8u, TX * 8u);
            // generic-proxy writes of the staging tile -> visible to the TMA store that the last
            // warp issues after the next barrier (the next tile's sweep barrier, or the one below)
            ptx::fence_proxy_async_smem();
        }
    }
    // x of the last tile; the staging tile must outlive the store
    if (kStage != 1 && it > 0) {
        __syncthreads();
        if (issue_lane >= 0) {
            store_x(tile_of(it - 1));
            asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
        }
    }
}

// ------------------------------------------------------------------------------------------
// Host side
// ------------------------------------------------------------------------------------------
inline bool is_pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }

// Leaf sizes the kernel is instantiated for: powers of two and 3, 5 times a power of two, so that
// line lengths 2^k, 3 * 2^k and 5 * 2^k tile as CL x W x m0 with W a power of two.
constexpr int kLeafSizes[] = {16, 12, 10, 8, 6, 4, 2};

// Eligibility: nx even (TMA global strides are multiples of 16 B), the line tiles as CL x W x m0
// with CL and W powers of two (W <= 32: the tree of a line runs inside a warp), the tile fits
// shared memory.  The leaves need NOT nest with the paper's partitions (D1): every
// level of the recursion is a Schur complement of the same matrix, so cutting a line into leaves
// of m0 rows instead of partitions of ny/P rows changes x only by rounding.  When m0 divides
// ny/P with a power-of-two quotient, one tree level is exactly the paper's 2P-row reduced system.
inline bool configure_tma_fused(TmaFusedConfig *out, int nx, int ny, int P, int want_lines,
                                int want_cluster, int want_leaf, const cudaDeviceProp &prop,
                                const char **why, bool xaxis = false, bool zaxis = false, int want_slots = 0)
{
    (void)P;
    // x sweep: nx = number of lanes (caller's ny), ny = line length (caller's nx)
    if (xaxis) {
        if (ny % 2) { *why = "TMA path needs even nx (16-byte global strides)"; return false; }
        if ((want_lines && want_lines != 16) || (want_leaf && want_leaf != 16)) {
            *why = "x sweeps use 16 lines per tile and 16-row leaves"; return false;
        }
        want_lines = 16; want_leaf = 16;
    } else if (nx % 2) { *why = "TMA path needs even nx (16-byte global strides)"; return false; }
    const size_t max_smem = prop.sharedMemPerBlockOptin;
    const size_t sm_smem = prop.sharedMemPerMultiprocessor;
    TmaFusedConfig best; double best_score = -1.0;
    const int tx_opts[3] = {16, 32, 8};
    // clusters of 3 / 6 / 5: x sweeps of 3 * 2^k and 5 * 2^k cells (their leaves are whole 128-byte rows of 16 x,
    // so the odd factor cannot go into the leaf as it does for y / z sweeps)
    const int cl_opts[8] = {1, 2, 4, 8, 16, 3, 6, 5};
    for (int ti = 0; ti < 3; ++ti) {
        const int TX = tx_opts[ti];
        if (want_lines && TX != want_lines) continue;
        if (!want_lines && TX > 8 && nx < TX) continue;
        for (int ci = 0; ci < 8; ++ci) {
            const int CL = cl_opts[ci];
            if (want_cluster && CL != want_cluster) continue;
            if (CL > 8 && !want_cluster) continue;
            const bool odd_cl = CL == 3 || CL == 6 || CL == 5;
            if (ny % CL) continue;
            const int R = ny / CL;
            for (int m0 : kLeafSizes) {
                if (want_leaf && m0 != want_leaf) continue;
                if (m0 > R || R % m0 || !is_pow2(R / m0) || R / m0 > 32) continue;
                TmaFusedConfig c;
                c.lines = TX; c.cluster = CL; c.rows = R; c.leaf_rows = m0; c.leaves = R / m0;
                c.threads = c.leaves * TX;
                if (c.threads > 512 || (xaxis && c.threads > 256)) continue;
                // y / z sweeps of 3 * 2^k and 5 * 2^k rows: a cluster of 3, 6 or 5 that leaves 256 threads with
                // 16-row leaves (the tiling of the power-of-two lengths) beats leaves of 12 / 10 rows under a
                // power-of-two cluster (ny = 768: 6.12 against 5.24 TB/s, 1280: 5.48 against 3.79, 384: 6.26
                // against 5.53, 1536: 5.14 against 4.34); smaller CTAs do not (ny = 640, 128 threads: 3.1 against 4.7)
                if (odd_cl && !xaxis && want_cluster != CL && !(m0 == 16 && c.threads == 256)) continue;
                c.nlev = 0;
                while ((1 << c.nlev) < c.leaves) ++c.nlev;
                c.box_rows = R;
                while (c.box_rows > 256) c.box_rows /= 2;
                if (R % c.box_rows) continue;
                c.xaxis = xaxis;
                // as many ring slots (<= 8 = two whole tiles) as shared memory holds
                c.slots = 0;
                for (int na = want_slots ? want_slots : 8; na >= (want_slots ? want_slots : 4); --na) {
                    c.smem = tma_fused_smem_bytes(TX, R, c.leaves, CL, na, xaxis);
                    if (c.smem <= max_smem) { c.slots = na; break; }
                }
                if (!c.slots) continue;
                long ctas = (long)(sm_smem / (c.smem + 1024));
                const long launch_threads = (c.threads + 31) & ~31;
                const long by_thr = 2048 / launch_threads;
                if (by_thr < ctas) ctas = by_thr;
                if (ctas < 1) continue;
                // Measured on B200 (cfg 3 shapes): the tile period is set by the serial phases, so
                // long leaves (fewer tree levels) win first; then resident cells, small clusters,
                // 128 B row segments.  Registers per thread of the instantiation: launch_tma_m0.
                const long regs = c.threads > 256 ? 128 : 255;
                const long by_regs = 65536 / (regs * launch_threads);
                if (by_regs < ctas) ctas = by_regs;
                if (ctas < 1) continue;
                double cells = (double)ctas * R * TX;
                if (cells > 8192.0) cells = 8192.0;
                // 128 B row segments: with 64 B segments the persistent clusters drift apart in a
                // long run and DRAM row-buffer locality between neighbouring x tiles is lost
                // (measured: 4.4 -> 3.1 TB/s from 256 to 1024 slices at TX = 8, flat at TX = 16)
                double score = 10000.0 * m0 + cells + (c.threads >= 32 ? 4000.0 : 0.0) + (c.slots > 4 ? 500.0 : 0.0) -
                               50.0 * CL - (c.threads > 256 && m0 > 8 ? 60000.0 : 0.0) +   // 128 registers: spills
                               // z sweeps: rows of a line are whole slices apart (a DRAM page and a
                               // TLB entry per row), 256 B segments pay (0.99 -> 0.91 ms on cfg 4)
                               (zaxis ? (TX == 32 ? 3000.0 : (TX == 16 ? 1000.0 : 0.0))
                                      : (TX == 16 ? 3000.0 : (TX == 32 ? 1000.0 : 0.0)));
                if (score > best_score) { best_score = score; best = c; }
            }
        }
    }
    if (best_score < 0) {
        *why = "no (lines, cluster, leaf) tiling with a power-of-two tree of <= 32 leaves fits shared memory";
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
                                 long long rs, long long os, bool axis_z, int TX, int box_rows, bool pair = false)
{
    tdma_encode_tiled_fn enc = get_encode_tiled();
    if (!enc) return false;
    cuuint64_t gdim[3] = {(cuuint64_t)nx, (cuuint64_t)(axis_z ? nslices : nrows), (cuuint64_t)(axis_z ? nrows : nslices)};
    cuuint64_t gstr[2] = {(cuuint64_t)(axis_z ? os : rs) * sizeof(double), (cuuint64_t)(axis_z ? rs : os) * sizeof(double)};
    cuuint32_t box[3] = {(cuuint32_t)TX, (cuuint32_t)(axis_z ? 1 : box_rows), (cuuint32_t)(axis_z ? box_rows : 1)};
    cuuint32_t estr[3] = {1, 1, 1};
    const size_t inner = (size_t)TX * sizeof(double);   // one L2 request per row segment, no over-fetch
    const CUtensorMapL2promotion promo = inner >= 256 ? CU_TENSOR_MAP_L2_PROMOTION_L2_256B
                                       : (inner >= 128 || pair) ? CU_TENSOR_MAP_L2_PROMOTION_L2_128B
                                                      : CU_TENSOR_MAP_L2_PROMOTION_L2_64B;
    return enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<void *>(base), gdim, gstr, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, promo,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// x sweep: contiguous fp64 slab (rows = x fastest, lanes = y, slices) viewed as the 4-D tensor
// (16 x, lanes, nrows / 16 leaves, slices); box (16, TX, W, 1) with the 128-byte swizzle: one copy per
// array and tile, landing as [leaf][line][16 x].  (The leaf dimension has the SMALLER stride, 128 B,
// than the lane dimension before it; tensor maps do not require ordered strides.)
inline bool make_xsweep_tensor_map(CUtensorMap *tm, const void *base, int nrows, int nlanes, int nslices, int TX, int W)
{
    tdma_encode_tiled_fn enc = get_encode_tiled();
    if (!enc || nrows % 16) return false;
    cuuint64_t gdim[4] = {16, (cuuint64_t)nlanes, (cuuint64_t)(nrows / 16), (cuuint64_t)nslices};
    cuuint64_t gstr[3] = {(cuuint64_t)nrows * sizeof(double), 128, (cuuint64_t)nrows * nlanes * sizeof(double)};
    cuuint32_t box[4] = {16, (cuuint32_t)TX, (cuuint32_t)W, 1};
    cuuint32_t estr[4] = {1, 1, 1, 1};
    return enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<void *>(base), gdim, gstr, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int TX, int M0, bool kCluster, int MAXT, bool kX = false, int kStage = 0>
inline cudaError_t launch_tma_inst(TmaFusedConfig &cfg, const CUtensorMap *tm, const TmaFusedParams &prm,
                                   cudaStream_t st)
{
    auto kern = fused_tma_kernel<TX, M0, kCluster, MAXT, kX, kStage>;
    const size_t smem_bytes = cfg.smem;
    cudaLaunchConfig_t lc = {};
    lc.blockDim = dim3((cfg.threads + 31) & ~31);
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
            e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kern, (int)lc.blockDim.x, smem_bytes);
            if (e != cudaSuccess) return e;
            n *= sms;
            if (kStage != 0) n /= cfg.cluster;          // groups of `cluster` independent CTAs per line tile
        }
        if (n < 1) return cudaErrorLaunchOutOfResources;
        cfg.max_clusters = n;
    }
    if (prm.ntiles <= 0) return cudaSuccess;    // prepare only (attributes + persistent grid size)
    const int nc = prm.ntiles < cfg.max_clusters ? prm.ntiles : cfg.max_clusters;
    lc.gridDim = dim3((unsigned)(nc * cfg.cluster));
    return cudaLaunchKernelEx(&lc, kern, tm[0], tm[1], tm[2], tm[3], tm[4], prm);
}

// The dispatch over every instantiation of the fused solve: only the plan's translation unit wants
// them compiled (the other units instantiate their own kernels from the template above).
#ifdef TDMA_FUSED_TMA_DISPATCH
template <int TX, int M0, bool kCluster>
inline cudaError_t launch_tma_m0(TmaFusedConfig &cfg, const CUtensorMap *tm, const TmaFusedParams &prm,
                                 cudaStream_t st)
{
    // registers: the parked interior rows take 6 (M0 - 2) of them; <= 256 threads leave 255 per
    // thread, <= 512 leave 128
    if (cfg.threads <= 256) return launch_tma_inst<TX, M0, kCluster, 256>(cfg, tm, prm, st);
    return launch_tma_inst<TX, M0, kCluster, 512>(cfg, tm, prm, st);
}

template <int TX, bool kCluster>
cudaError_t launch_tma_tx(TmaFusedConfig &cfg, const CUtensorMap *tm, const TmaFusedParams &prm, cudaStream_t st)
{
    switch (cfg.leaf_rows) {
    case 2: return launch_tma_m0<TX, 2, kCluster>(cfg, tm, prm, st);
    case 4: return launch_tma_m0<TX, 4, kCluster>(cfg, tm, prm, st);
    case 6: return launch_tma_m0<TX, 6, kCluster>(cfg, tm, prm, st);
    case 8: return launch_tma_m0<TX, 8, kCluster>(cfg, tm, prm, st);
    case 10: return launch_tma_m0<TX, 10, kCluster>(cfg, tm, prm, st);
    case 12: return launch_tma_m0<TX, 12, kCluster>(cfg, tm, prm, st);
    case 16: return launch_tma_m0<TX, 16, kCluster>(cfg, tm, prm, st);
    default: return cudaErrorInvalidValue;
    }
}

// a, b, c, d, x: batch base pointers (slice 0 of the launch), 16-byte aligned.
inline cudaError_t launch_tma_fused(TmaFusedConfig &cfg, const double *a, const double *b,
                                    const double *c, const double *d, double *x, int nx, int ny,
                                    int nzs, long long rs, long long os, bool axis_z, bool periodic,
                                    cudaStream_t st)
{
    const void *ptr[5] = {a, b, c, d, x};
    const int xtiles = (nx + cfg.lines - 1) / cfg.lines;
    // 64-byte row segments: neighbouring x tiles share 128-byte lines -> a cluster takes them in pairs
    const bool pair = !cfg.xaxis && cfg.lines * sizeof(double) < 128 && xtiles % 2 == 0;
    CUtensorMap dummy[5];
    const CUtensorMap *tm = dummy;
    if (nzs > 0) {              // everything else a map depends on is fixed per plan
        TmaFusedConfig::MapSet *hit = nullptr;
        for (int i = 0; i < cfg.nmaps && !hit; ++i) {
            TmaFusedConfig::MapSet &m = cfg.maps[i];
            if (m.nzs == nzs && m.ptr[0] == a && m.ptr[1] == b && m.ptr[2] == c && m.ptr[3] == d && m.ptr[4] == x) hit = &m;
        }
        if (!hit) {
            TmaFusedConfig::MapSet &m = cfg.maps[cfg.next_map];
            for (int i = 0; i < 5; ++i) {
                if (cfg.xaxis ? !make_xsweep_tensor_map(&m.tm[i], ptr[i], ny, nx, nzs, cfg.lines, cfg.leaves)
                              : !make_slab_tensor_map(&m.tm[i], ptr[i], nx, ny, nzs, rs, os, axis_z, cfg.lines, cfg.box_rows, pair)) {
                    m.nzs = -1;
                    return cudaErrorInvalidValue;
                }
                m.ptr[i] = ptr[i];
            }
            m.nzs = nzs;
            cfg.next_map = (cfg.next_map + 1) % TmaFusedConfig::kMapSets;
            if (cfg.nmaps < TmaFusedConfig::kMapSets) ++cfg.nmaps;
            hit = &m;
        }
        tm = hit->tm;
    }
    TmaFusedParams prm;
    prm.nx = nx; prm.ny = ny; prm.nzs = nzs;
    prm.x = x;
    prm.rs = rs; prm.os = os; prm.axis_z = axis_z ? 1 : 0; prm.periodic = periodic ? 1 : 0;
    prm.CL = cfg.cluster; prm.R = cfg.rows; prm.W = cfg.leaves; prm.NS = cfg.slots;
    prm.xtiles = xtiles;
    prm.ntiles = prm.xtiles * nzs;
    prm.pair = pair ? 1 : 0;
    prm.box_rows = cfg.box_rows; prm.nbox = cfg.rows / cfg.box_rows;
    const bool cl = cfg.cluster > 1;
    if (cfg.xaxis)
        return cl ? launch_tma_inst<16, 16, true, 256, true>(cfg, tm, prm, st)
                  : launch_tma_inst<16, 16, false, 256, true>(cfg, tm, prm, st);
    switch (cfg.lines) {
    case 32: return cl ? launch_tma_tx<32, true>(cfg, tm, prm, st) : launch_tma_tx<32, false>(cfg, tm, prm, st);
    case 16: return cl ? launch_tma_tx<16, true>(cfg, tm, prm, st) : launch_tma_tx<16, false>(cfg, tm, prm, st);
    case 8: return cl ? launch_tma_tx<8, true>(cfg, tm, prm, st) : launch_tma_tx<8, false>(cfg, tm, prm, st);
    default: return cudaErrorInvalidValue;
    }
}

#endif  // TDMA_FUSED_TMA_DISPATCH

}  // namespace tdma
