// FUSED variant (sm_100a): the divide-and-conquer solve of PAPER.md:49-58 inside ONE kernel, the
// recursion mapped onto the B200 hierarchy  thread -> CTA (shared memory) -> cluster (DSMEM).
//
// Mapping of the paper's objects:
//   processor / rank      -> CTA of a thread-block cluster; CTA c owns rows
//                                              c*R .. c*R+R-1 (R = ny/CL) of TX consecutive lines
//   Stage A "solve the decoupled system"    -> the paper calls a parallel library solver here
//                        (cuSPARSE CR-PCR); we recurse instead: every
//                                              partition of m = ny/P rows is cut into leaves of m0
//                                              rows, one THREAD per (line, leaf) runs the modified
//                                              Thomas reduction from HBM (a, b, c, d read once),
//                                              then one thread per (line, partition) reduces the
//                                              2*(m/m0) leaf boundary equations to the partition's
//                                              two boundary equations  (= rows 2p, 2p+1 of the
//                                              paper's reduced system)
//   forward-eliminated rows / spikes         -> stay in SHARED MEMORY (24 B/cell), never in HBM
//   send_A / MPI_Alltoall / recv_B           -> distributed-shared-memory stores: every CTA
//                  writes its boundary equations straight into the
//                                              smem of the CTA that solves that line
//   even distribution of stage B [16]        -> CTA c solves the reduced systems of lines
//                            c*TX/CL .. (c+1)*TX/CL - 1   (Thomas, unit diagonal)
//   top = 1: the 2P-row reduced system is exchanged as is (literal stage B);
//   top = 2: each CTA first reduces its 2*P/CL rows further to 2 rows (same recursion), the
//            cluster exchanges / solves 2*CL rows
//   send_B / Alltoall / recv_C               -> DSMEM stores of the boundary values back into the
//                                              owning CTA's smem
//   Stage C                   -> top-down back-substitution from shared memory,
//                                              x streamed to HBM
// HBM traffic: a, b, c, d read once, x written once = 40 B/cell.
//
// In-place storage.  A node of the recursion (leaf, partition, ...) spans `span` consecutive rows
// of the CTA's tile and is represented by two equations with unit diagonal,
//        first-row eq:  A x_prev_last + x_first + C x_last       = D
//        last-row  eq:  A x_first     + x_last  + C x_next_first = D,
// kept in the smem slots of the node's first and last row.  Row q of a level (q = 0, 1, 2, ...
// = first, last, first, last ... of consecutive nodes) therefore lives at tile row
//        pos(q) = (q >> 1) * span + (q & 1) * (span - 1).
// Reducing a group of g such rows (one thread per line and group, serial in q) overwrites rows
// 1 .. g-2 with their forward-eliminated form  a' x_first + x_q + c' x_{q+1} = d'  and leaves the
// group's own two equations in rows 0 and g-1, which are exactly the next level's slots.
// Back-substitution walks the levels in reverse, overwriting d' with x.
#pragma once
#include <cooperative_groups.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "tdma_stage_kernels.cuh"

namespace tdma {

namespace cg = cooperative_groups;

constexpr int kMaxFusedLevels = 6;

struct FusedConfig {
    int lines = 0;         // TX: lines (x extent) per cluster tile
    int cluster = 0;       // CL: CTAs per cluster
    int rows = 0;          // R = ny / CL rows per CTA
    int leaf_rows = 0;     // m0
    int leaves = 0;        // W = R / m0 leaves per CTA and line
    int threads = 0;       // W * TX
    int lines_solved = 0;  // TXS = TX / CL top systems solved per CTA
    int top_mode = 0;      // 1 = partition level (2P rows), 2 = CTA level (2 CL rows)
    int nlev = 0;          // in-CTA reduction levels above the leaves
    int lev_g[kMaxFusedLevels] = {};       // rows per group
    int lev_groups[kMaxFusedLevels] = {};  // groups per CTA
    int lev_span[kMaxFusedLevels] = {};    // span (tile rows) of the level's input nodes
    int top_nodes = 0;     // nodes per CTA handed to the cluster-level solve
    int top_span = 0;      // their span
    size_t smem = 0;
};

struct FusedParams {
    const double *a, *b, *c, *d;
    double *x;
    int nx, ny, nzs;
    int CL, R, m0, W, TXS;
    int nlev;
    int lev_g[kMaxFusedLevels], lev_groups[kMaxFusedLevels], lev_span[kMaxFusedLevels];
    int top_nodes, top_span;
    int xtiles;  // ceil(nx / TX)
};

__host__ __device__ inline size_t fused_smem_bytes(int TX, int R, int CL, int top_nodes)
{
    const int TXS = TX / CL;
    return ((size_t)3 * R * TX                              // rows: [R][3][TX]
            + (size_t)4 * 2 * top_nodes * CL * TXS)         // top system RA, RC, RD + c' column
           * sizeof(double);
}

__device__ __forceinline__ int node_pos(int q, int span) { return (q >> 1) * span + (q & 1) * (span - 1); }

// TX: lines per tile (compile time: smem offsets become immediates).  MAXT / MINB: launch bounds
// (register budget).  U: rows of a, b, c, d kept in flight per thread.
template <int TX, bool kCluster, int MAXT, int MINB, int U>
__global__ void __launch_bounds__(MAXT, MINB) fused_kernel(const FusedParams prm)
{
    extern __shared__ __align__(16) double smem[];
    constexpr int ROW = 3 * TX;           // doubles per tile row: a' | c' | d'
    const int R = prm.R, m0 = prm.m0, CL = prm.CL, TXS = prm.TXS;
    double *__restrict__ rows = smem;                       // [R][3][TX]
    double *__restrict__ red = smem + (size_t)R * ROW;      // [4][NTR][TXS]
    const int ntr_cta = 2 * prm.top_nodes;                  // top rows contributed per CTA
    const int NTR = ntr_cta * CL;                           // top rows per line

    unsigned crank = 0;
    if (kCluster) crank = cg::this_cluster().block_rank();
    const int tile = blockIdx.x / CL;
    const int xt = tile % prm.xtiles;
    const int k = tile / prm.xtiles;
    const int t = threadIdx.x;
    const int lx = t % TX, leaf = t / TX;
    const int nx = prm.nx;
    const int x0 = xt * TX;
    const bool active = x0 + lx < nx;                       // ragged x tail: lane computes a copy
    const int gx = active ? x0 + lx : nx - 1;
    const int r0 = leaf * m0;                               // leaf's first tile row
    const int grow0 = (int)crank * R + r0;                  // ... and global row
    const size_t off0 = ((size_t)k * prm.ny + grow0) * (size_t)nx + gx;
    const unsigned s = (unsigned)nx;
    // split-phase cluster barrier: every CTA of the cluster must have started before the first
    // distributed-shared-memory store; the matching wait sits right before the A2B loop
    if (kCluster) asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");

    // ---------------- leaves: modified Thomas reduction straight from HBM ----------------
    {
        const double *__restrict__ a = prm.a + off0;
        const double *__restrict__ b = prm.b + off0;
        const double *__restrict__ c = prm.c + off0;
        const double *__restrict__ d = prm.d + off0;
        const bool first_leaf = (grow0 == 0), last_leaf = (grow0 + m0 == prm.ny);
        double *__restrict__ tr = rows + (size_t)r0 * ROW + lx;

        // first-row equation  fa x_{-1} + fb x_0 + fc x_frontier = fd
        double inv = 1.0 / ld_stream(b);
        double fa = first_leaf ? 0.0 : ld_stream(a) * inv;
        double fc = ld_stream(c) * inv;
        double fd = ld_stream(d) * inv;
        double fb = 1.0;
        // row 1 in forward form  pa x_0 + x_1 + pc x_2 = pd
        double pa, pc, pd;
        {
            const double a1 = ld_stream(a + s), b1 = ld_stream(b + s);
            double c1 = ld_stream(c + s);
            const double d1 = ld_stream(d + s);
            if (last_leaf && m0 == 2) c1 = 0.0;
            inv = 1.0 / b1;
            pa = a1 * inv; pc = c1 * inv; pd = d1 * inv;
        }
        double qa[U], qb[U], qc[U], qd[U];
        unsigned o = 2 * s;                                  // element offset of the next row to load
#pragma unroll
        for (int u = 0; u < U; ++u) {
            if (2 + u < m0) {
                qa[u] = ld_stream(a + o); qb[u] = ld_stream(b + o);
                qc[u] = ld_stream(c + o); qd[u] = ld_stream(d + o);
                o += s;
            }
        }
        for (int rb = 2; rb < m0; rb += U) {
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int r = rb + u;
                if (r < m0) {
                    const double ar = qa[u], br = qb[u], dr = qd[u];
                    const double cr = (last_leaf && r == m0 - 1) ? 0.0 : qc[u];
                    if (r + U < m0) {                        // refill the slot: row r + U
                        qa[u] = ld_stream(a + o); qb[u] = ld_stream(b + o);
                        qc[u] = ld_stream(c + o); qd[u] = ld_stream(d + o);
                        o += s;
                    }
                    // fold row r-1 into the first-row equation, park it for back-substitution
                    fb = fma(-fc, pa, fb);
                    fd = fma(-fc, pd, fd);
                    fc = -fc * pc;
                    double *w = tr + (size_t)(r - 1) * ROW;
                    w[0] = pa; w[TX] = pc; w[2 * TX] = pd;
                    inv = 1.0 / fma(-ar, pc, br);
                    pd = fma(-ar, pd, dr) * inv;
                    pc = cr * inv;
                    pa = -(ar * pa) * inv;
                }
            }
        }
        inv = 1.0 / fb;                                      // m0 == 2: fb = 1, frontier is x_1
        tr[0] = fa * inv; tr[TX] = fc * inv; tr[2 * TX] = fd * inv;
        double *w = tr + (size_t)(m0 - 1) * ROW;
        w[0] = pa; w[TX] = pc; w[2 * TX] = pd;
    }

    // ---------------- in-CTA levels: groups of boundary equations -> two equations ---------
    for (int lv = 0; lv < prm.nlev; ++lv) {
        __syncthreads();
        const int g = prm.lev_g[lv], span = prm.lev_span[lv];
        if (leaf < prm.lev_groups[lv]) {
            const int q0 = leaf * g;
            double *__restrict__ base = rows + lx;
            double *p0 = base + (size_t)node_pos(q0, span) * ROW;
            double *p1 = base + (size_t)node_pos(q0 + 1, span) * ROW;
            double fa = p0[0], fc = p0[TX], fd = p0[2 * TX], fb = 1.0;
            double pa = p1[0], pc = p1[TX], pd = p1[2 * TX];
            double *prev = p1;
            double *cur = base + (size_t)node_pos(q0 + 2, span) * ROW;
            double aq = cur[0], cq = cur[TX], dq = cur[2 * TX];
            for (int q = 2; q < g; ++q) {
                double *nxt = cur;
                double an = 0.0, cn = 0.0, dn = 0.0;
                if (q + 1 < g) {                             // next row's loads go out first
                    nxt = base + (size_t)node_pos(q0 + q + 1, span) * ROW;
                    an = nxt[0]; cn = nxt[TX]; dn = nxt[2 * TX];
                }
                fb = fma(-fc, pa, fb);
                fd = fma(-fc, pd, fd);
                fc = -fc * pc;
                prev[0] = pa; prev[TX] = pc; prev[2 * TX] = pd;
                const double inv = 1.0 / fma(-aq, pc, 1.0);
                pd = fma(-aq, pd, dq) * inv;
                pc = cq * inv;
                pa = -(aq * pa) * inv;
                prev = cur; cur = nxt; aq = an; cq = cn; dq = dn;
            }
            const double inv = 1.0 / fb;
            p0[0] = fa * inv; p0[TX] = fc * inv; p0[2 * TX] = fd * inv;
            prev[0] = pa; prev[TX] = pc; prev[2 * TX] = pd;
        }
    }

    // ---------------- A2B: top-level equations -> smem of the CTA that solves the line ------
    __syncthreads();
    if (kCluster) asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
    {
        const size_t plane = (size_t)NTR * TXS;
        for (int e = t; e < ntr_cta * TX; e += blockDim.x) {
            const int j = e / TX, l = e - j * TX;
            const double *src = rows + (size_t)node_pos(j, prm.top_span) * ROW + l;
            const int owner = l / TXS, col = l - owner * TXS;
            double *dst = red;
            if (kCluster) dst = cg::this_cluster().map_shared_rank(red, owner);
            const size_t q = (size_t)((int)crank * ntr_cta + j) * TXS + col;
            dst[q] = src[0]; dst[plane + q] = src[TX]; dst[2 * plane + q] = src[2 * TX];
        }
    }
    if (kCluster) cg::this_cluster().sync(); else __syncthreads();

    // ---------------- Stage B: Thomas on the NTR-row top system of my TXS lines -------------
    if (t < TXS) {
        const size_t plane = (size_t)NTR * TXS;
        const double *ra = red + t, *rc = red + plane + t;
        double *yv = red + 2 * plane + t;                    // d' then y, in place
        double *cpw = red + 3 * plane + t;
        double cp = rc[0], dp = yv[0];
        cpw[0] = cp;
        double an = 0.0, cn = 0.0, dn = 0.0;
        if (NTR > 1) { an = ra[TXS]; cn = rc[TXS]; dn = yv[TXS]; }
        for (int q = 1; q < NTR; ++q) {
            const double aq = an, cq = cn, dq = dn;
            if (q + 1 < NTR) {
                an = ra[(size_t)(q + 1) * TXS]; cn = rc[(size_t)(q + 1) * TXS]; dn = yv[(size_t)(q + 1) * TXS];
            }
            const double inv = 1.0 / fma(-aq, cp, 1.0);
            dp = fma(-aq, dp, dq) * inv;
            cp = cq * inv;
            cpw[(size_t)q * TXS] = cp;
            yv[(size_t)q * TXS] = dp;
        }
        // backward + B2C: boundary values go into the d' slot of the owning CTA's tile row
        const int line = (int)crank * TXS + t;
        double xq = dp;
        for (int q = NTR - 1; q >= 0; --q) {
            if (q < NTR - 1) xq = fma(-cpw[(size_t)q * TXS], xq, yv[(size_t)q * TXS]);
            const int dest = q / ntr_cta, j = q - dest * ntr_cta;
            double *rdst = rows;
            if (kCluster) rdst = cg::this_cluster().map_shared_rank(rows, dest);
            rdst[(size_t)node_pos(j, prm.top_span) * ROW + 2 * TX + line] = xq;
        }
    }
    if (kCluster) cg::this_cluster().sync(); else __syncthreads();

    // ---------------- back-substitution, top-down through the in-CTA levels ----------------
    for (int lv = prm.nlev - 1; lv >= 0; --lv) {
        const int g = prm.lev_g[lv], span = prm.lev_span[lv];
        if (leaf < prm.lev_groups[lv]) {
            const int q0 = leaf * g;
            double *__restrict__ base = rows + lx;
            const double xf = base[(size_t)node_pos(q0, span) * ROW + 2 * TX];
            double xn = base[(size_t)node_pos(q0 + g - 1, span) * ROW + 2 * TX];
            for (int q = g - 2; q >= 1; --q) {
                double *p = base + (size_t)node_pos(q0 + q, span) * ROW;
                xn = fma(-p[TX], xn, fma(-p[0], xf, p[2 * TX]));
                p[2 * TX] = xn;
            }
        }
        __syncthreads();
    }

    // ---------------- leaves: back-substitution from shared memory, x streamed to HBM ------
    {
        const double *__restrict__ tr = rows + (size_t)r0 * ROW + lx;
        double *__restrict__ x = prm.x + off0;
        const double xf = tr[2 * TX];
        const double xl = tr[(size_t)(m0 - 1) * ROW + 2 * TX];
        if (active) {
            st_stream(x, xf);
            st_stream(x + (size_t)(m0 - 1) * s, xl);
        }
        double xn = xl;
        const double *p = tr + (size_t)(m0 - 2) * ROW;
        unsigned o = (unsigned)(m0 - 2) * s;
#pragma unroll 4
        for (int r = m0 - 2; r >= 1; --r) {
            xn = fma(-p[TX], xn, fma(-p[0], xf, p[2 * TX]));
            if (active) st_stream(x + o, xn);
            p -= ROW; o -= s;
        }
    }
}

// ------------------------------------------------------------------------------------------
// Host side: choose (TX, CL, m0, levels) and launch.
// ------------------------------------------------------------------------------------------
inline int smallest_divisor_at_least(int n, int lo)
{
    for (int k = lo < 1 ? 1 : lo; k <= n; ++k)
        if (n % k == 0) return k;
    return n;
}

// Level table above the leaves (mirrors the derivation at the top of this file).
inline bool build_levels(FusedConfig *cfg, int ny, int P)
{
    const int m = ny / P, m0 = cfg->leaf_rows, s = m / m0;
    int nodes = cfg->leaves, span = m0, n = 0;
    if (s > 1) {                       // leaves -> partitions (the paper's stage A output)
        cfg->lev_g[n] = 2 * s; cfg->lev_groups[n] = nodes / s; cfg->lev_span[n] = span;
        ++n; nodes /= s; span *= s;
    }
    if (cfg->top_mode == 2) {          // partitions -> one node per CTA, fan-in <= 4 nodes
        while (nodes > 1) {
            if (n >= kMaxFusedLevels) return false;
            const int f = smallest_divisor_at_least(nodes, nodes < 4 ? nodes : 4);
            cfg->lev_g[n] = 2 * f; cfg->lev_groups[n] = nodes / f; cfg->lev_span[n] = span;
            ++n; nodes /= f; span *= f;
        }
    }
    cfg->nlev = n; cfg->top_nodes = nodes; cfg->top_span = span;
    return true;
}

// Pick TX / CL / m0.  Goal: about 512 resident threads per SM at <= 128 registers each (the
// leaf recurrences are latency bound: one division chain per thread), two or more CTAs per SM so
// that one tile's reduced solve overlaps another tile's HBM phase, row segments of 256 B.
inline bool configure_fused(FusedConfig *out, int nx, int ny, int P, int want_lines, int want_cluster,
                            int want_leaf, int want_top, const cudaDeviceProp &prop, const char **why)
{
    const int m = ny / P;
    const size_t max_smem = prop.sharedMemPerBlockOptin;
    const size_t sm_smem = prop.sharedMemPerMultiprocessor;
    int TX = want_lines;
    if (TX == 0) TX = nx >= 32 ? 32 : (nx >= 16 ? 16 : 8);
    if (TX != 8 && TX != 16 && TX != 32) { *why = "fused_lines must be 8, 16 or 32"; return false; }
    FusedConfig best; long best_score = -1;
    const int cl_opts[5] = {1, 2, 4, 8, 16};
    for (int ci = 0; ci < 5; ++ci) {
        const int CL = cl_opts[ci];
        if (want_cluster && CL != want_cluster) continue;
        if (CL > 8 && !want_cluster) continue;               // 16 is non-portable: only on request
        if (P % CL || TX % CL) continue;
        const int R = ny / CL;
        for (int m0 = 2; m0 <= m; ++m0) {
            if (m % m0) continue;
            if (want_leaf && m0 != want_leaf) continue;
            FusedConfig c;
            c.lines = TX; c.cluster = CL; c.rows = R; c.leaf_rows = m0; c.leaves = R / m0;
            c.threads = c.leaves * TX; c.lines_solved = TX / CL;
            if (c.threads > 1024) continue;
            c.top_mode = want_top ? want_top : 2;
            if (CL == 1 && P == 1) c.top_mode = 2;
            if (!build_levels(&c, ny, P)) continue;
            c.smem = fused_smem_bytes(TX, R, CL, c.top_nodes);
            if (c.smem > max_smem) continue;
            const int regs = c.threads <= 256 ? 128 : (c.threads <= 512 ? 128 : 64);
            long by_smem = (long)(sm_smem / (c.smem + 1024));
            long by_regs = 65536 / ((long)c.threads * regs);
            long by_thr = 2048 / c.threads;
            long ctas = by_smem < by_regs ? by_smem : by_regs;
            if (by_thr < ctas) ctas = by_thr;
            if (ctas < 1) continue;
            long resident = ctas * c.threads;
            if (resident > 512) resident = 512;
            // resident threads first, then >= 2 CTAs per SM, then longer leaves (less tree work),
            // then the smaller cluster
            long score = resident * 1000000L + (ctas >= 2 ? 100000L : 0) + (m0 >= 8 ? 10000L : 0) +
                         (long)(m0 > 64 ? 64 : m0) * 100L + (16 - CL);
            if (c.threads > 512) score -= 300L * 1000000L;   // 64-register kernels spill
            if (score > best_score) { best_score = score; best = c; }
        }
    }
    if (best_score < 0) {
        *why = "no (lines, cluster, leaf) choice fits shared memory / divisibility (P % cluster, 2^k lines)";
        return false;
    }
    *out = best;
    return true;
}

template <int TX, bool kCluster, int MAXT, int MINB, int U>
inline cudaError_t launch_fused_inst(const FusedConfig &cfg, const FusedParams &prm, cudaStream_t st)
{
    auto kern = fused_kernel<TX, kCluster, MAXT, MINB, U>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cfg.smem);
    if (e != cudaSuccess) return e;
    if (cfg.cluster > 8) {
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        if (e != cudaSuccess) return e;
    }
    cudaLaunchConfig_t lc = {};
    lc.gridDim = dim3((unsigned)((size_t)prm.xtiles * prm.nzs * cfg.cluster));
    lc.blockDim = dim3(cfg.threads);
    lc.dynamicSmemBytes = cfg.smem;
    lc.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = cfg.cluster; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    lc.attrs = attr;
    lc.numAttrs = kCluster ? 1 : 0;
    return cudaLaunchKernelEx(&lc, kern, prm);
}

template <int TX, bool kCluster>
inline cudaError_t launch_fused_tx(const FusedConfig &cfg, const FusedParams &prm, cudaStream_t st)
{
    if (cfg.threads <= 256) return launch_fused_inst<TX, kCluster, 256, 2, 4>(cfg, prm, st);
    if (cfg.threads <= 512) return launch_fused_inst<TX, kCluster, 512, 1, 4>(cfg, prm, st);
    return launch_fused_inst<TX, kCluster, 1024, 1, 2>(cfg, prm, st);
}

inline cudaError_t launch_fused(const FusedConfig &cfg, const double *a, const double *b,
                                const double *c, const double *d, double *x, int nx, int ny,
                                int nzs, cudaStream_t st)
{
    FusedParams prm;
    prm.a = a; prm.b = b; prm.c = c; prm.d = d; prm.x = x;
    prm.nx = nx; prm.ny = ny; prm.nzs = nzs;
    prm.CL = cfg.cluster; prm.R = cfg.rows; prm.m0 = cfg.leaf_rows; prm.W = cfg.leaves;
    prm.TXS = cfg.lines_solved; prm.nlev = cfg.nlev;
    for (int i = 0; i < kMaxFusedLevels; ++i) {
        prm.lev_g[i] = cfg.lev_g[i]; prm.lev_groups[i] = cfg.lev_groups[i]; prm.lev_span[i] = cfg.lev_span[i];
    }
    prm.top_nodes = cfg.top_nodes; prm.top_span = cfg.top_span;
    prm.xtiles = (nx + cfg.lines - 1) / cfg.lines;
    const bool cl = cfg.cluster > 1;
    switch (cfg.lines) {
    case 32: return cl ? launch_fused_tx<32, true>(cfg, prm, st) : launch_fused_tx<32, false>(cfg, prm, st);
    case 16: return cl ? launch_fused_tx<16, true>(cfg, prm, st) : launch_fused_tx<16, false>(cfg, prm, st);
    case 8: return cl ? launch_fused_tx<8, true>(cfg, prm, st) : launch_fused_tx<8, false>(cfg, prm, st);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace tdma
