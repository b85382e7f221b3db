// FUSED variant (sm_100a): the divide-and-conquer solve of PAPER.md:49-58 inside one kernel.
//
// Mapping of the paper's objects onto one GPU:
//   processor / rank p   -> CTA of a thread-block cluster; CTA c owns the
//                                             partitions c*PP .. c*PP+PP-1 (rows c*PP*m ..) of
//                                             TX consecutive lines
//   Stage A result x~, spikes-> forward-eliminated rows (a', c', d') kept in the
//                                             CTA's SHARED MEMORY (24 B/cell), never in HBM
//   send_A / MPI_Alltoall / recv_B          -> distributed-shared-memory stores: every CTA
//                  writes its boundary equations straight into the
//                                             smem of the CTA that solves that line
//   even distribution of stage B [16]       -> CTA c solves the reduced systems of lines
//                            c*TX/CL .. (c+1)*TX/CL - 1
//   send_B / Alltoall / recv_C              -> DSMEM stores of the 2 boundary values per
//                                             partition per line back to the owning CTA
//   Stage C                  -> back-substitution from shared memory, x streamed
//                                             to HBM
// HBM traffic: a, b, c, d read once, x written once = 40 B/cell.
#pragma once
#include <cooperative_groups.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "tdma_stage_kernels.cuh"

namespace tdma {

namespace cg = cooperative_groups;

struct FusedConfig {
    int lines = 0;    // TX: lines (x extent) per cluster tile
    int cluster = 0;  // CL: CTAs per cluster
    int pp = 0;       // partitions per CTA = P / CL
    int threads = 0;  // TX * PP
    int lines_solved = 0;  // TX / CL reduced systems solved per CTA
    size_t smem = 0;
};

struct FusedParams {
    const double *a, *b, *c, *d;
    double *x;
    int nx, ny, nzs, P, m, TX, PP, TXS;
    int xtiles;  // nx / TX
};

__host__ __device__ inline size_t fused_smem_doubles(int TX, int PP, int m, int P, int TXS)
{
    const size_t rows = (size_t)PP * m;
    return 3 * rows * TX          // forward-eliminated rows a', c', d'
           + 4 * (size_t)2 * P * TXS  // reduced system RA, RC, RD + Thomas c' work column
           + (size_t)2 * PP * TX;     // boundary values of my partitions (recv_C)
}

// MAXT bounds the CTA size (and with it the register budget), U = rows of a, b, c, d kept in
// flight per thread: few fat threads (long partitions) prefetch deep, many thin threads do not
// need to.
template <int CL, int MAXT, int U>
__global__ void __launch_bounds__(MAXT) fused_kernel(const FusedParams prm)
{
    extern __shared__ __align__(16) double smem[];
    const int TX = prm.TX, PP = prm.PP, m = prm.m, P = prm.P, TXS = prm.TXS;
    const int rows = PP * m;
    double *__restrict__ s_a = smem;
    double *__restrict__ s_c = s_a + (size_t)rows * TX;
    double *__restrict__ s_d = s_c + (size_t)rows * TX;
    double *red = s_d + (size_t)rows * TX;  // [4][2P][TXS]
    double *yl = red + (size_t)4 * 2 * P * TXS;  // [2PP][TX]

    unsigned crank = 0;
    if (CL > 1) crank = cg::this_cluster().block_rank();
    const int tile = blockIdx.x / CL;
    const int xt = tile % prm.xtiles;
    const int k = tile / prm.xtiles;
    const int t = threadIdx.x;
    const int lx = t % TX, lp = t / TX;
    const int p = (int)crank * PP + lp;
    const int nx = prm.nx;
    const size_t s = (size_t)nx;
    const size_t off0 = (size_t)k * prm.ny * s + (size_t)xt * TX + lx + (size_t)p * m * s;
    const bool first_part = (p == 0), last_part = (p == P - 1);

    // ---------------- Stage A: forward elimination, rows kept in shared memory -----------
    {
        const double *__restrict__ a = prm.a + off0;
        const double *__restrict__ b = prm.b + off0;
        const double *__restrict__ c = prm.c + off0;
        const double *__restrict__ d = prm.d + off0;
        double *__restrict__ ta = s_a + (size_t)lp * m * TX + lx;
        double *__restrict__ tc = s_c + (size_t)lp * m * TX + lx;
        double *__restrict__ td = s_d + (size_t)lp * m * TX + lx;

        double inv = 1.0 / ld_stream(b);
        double fa = first_part ? 0.0 : ld_stream(a) * inv;
        double fc = ld_stream(c) * inv;
        double fd = ld_stream(d) * inv;
        double fb = 1.0;
        double pa, pc, pd;
        {
            const double a1 = ld_stream(a + s), b1 = ld_stream(b + s);
            double c1 = ld_stream(c + s);
            const double d1 = ld_stream(d + s);
            if (last_part && m == 2) c1 = 0.0;
            inv = 1.0 / b1;
            pa = a1 * inv; pc = c1 * inv; pd = d1 * inv;
        }
        double na[U], nb[U], nc[U], nd[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int r = 2 + u;
            if (r < m) {
                na[u] = ld_stream(a + r * s); nb[u] = ld_stream(b + r * s);
                nc[u] = ld_stream(c + r * s); nd[u] = ld_stream(d + r * s);
            }
        }
        for (int r0 = 2; r0 < m; r0 += U) {
            double ca[U], cb[U], cc[U], cd[U];
#pragma unroll
            for (int u = 0; u < U; ++u) { ca[u] = na[u]; cb[u] = nb[u]; cc[u] = nc[u]; cd[u] = nd[u]; }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int r = r0 + U + u;
                if (r < m) {
                    na[u] = ld_stream(a + r * s); nb[u] = ld_stream(b + r * s);
                    nc[u] = ld_stream(c + r * s); nd[u] = ld_stream(d + r * s);
                }
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int r = r0 + u;
                if (r < m) {
                    fb = fma(-fc, pa, fb);
                    fd = fma(-fc, pd, fd);
                    fc = -fc * pc;
                    ta[(size_t)(r - 1) * TX] = pa;
                    tc[(size_t)(r - 1) * TX] = pc;
                    td[(size_t)(r - 1) * TX] = pd;
                    const double ar = ca[u];
                    const double cr = (last_part && r == m - 1) ? 0.0 : cc[u];
                    inv = 1.0 / fma(-ar, pc, cb[u]);
                    pd = fma(-ar, pd, cd[u]) * inv;
                    pc = cr * inv;
                    pa = -(ar * pa) * inv;
                }
            }
        }
        inv = 1.0 / fb;
        // ------------- A2B: boundary equations -> smem of the CTA that solves this line ----
        const int owner = lx / TXS, col = lx - owner * TXS;
        double *dst = red;
        if (CL > 1) dst = cg::this_cluster().map_shared_rank(red, owner);
        const size_t plane = (size_t)2 * P * TXS;
        const size_t q0 = (size_t)(2 * p) * TXS + col, q1 = q0 + TXS;
        dst[q0] = fa * inv; dst[plane + q0] = fc * inv; dst[2 * plane + q0] = fd * inv;
        dst[q1] = pa;       dst[plane + q1] = pc;       dst[2 * plane + q1] = pd;
    }
    if (CL > 1) cg::this_cluster().sync(); else __syncthreads();

    // ---------------- Stage B: reduced 2P-row systems of my TXS lines --------------------
    if (t < TXS) {
        const int Q = 2 * P;
        const size_t plane = (size_t)Q * TXS;
        const double *ra = red + t, *rc = red + plane + t, *rd = red + 2 * plane + t;
        double *cpw = red + 3 * plane + t;
        double cp = rc[0], dp = rd[0];
        cpw[0] = cp;
        // forward; y is kept in the rd column
        double *yv = red + 2 * plane + t;
        for (int q = 1; q < Q; ++q) {
            const double aq = ra[(size_t)q * TXS];
            const double inv = 1.0 / fma(-aq, cp, 1.0);
            dp = fma(-aq, dp, rd[(size_t)q * TXS]) * inv;
            cp = rc[(size_t)q * TXS] * inv;
            cpw[(size_t)q * TXS] = cp;
            yv[(size_t)q * TXS] = dp;
        }
        // backward + B2C: boundary values go to the CTA that owns the partition
        const int line = (int)crank * TXS + t;
        double xq = dp;
        for (int q = Q - 1; q >= 0; --q) {
            if (q < Q - 1) xq = fma(-cpw[(size_t)q * TXS], xq, yv[(size_t)q * TXS]);
            const int pq = q >> 1;
            const int dest = pq / PP;
            double *ydst = yl;
            if (CL > 1) ydst = cg::this_cluster().map_shared_rank(yl, dest);
            ydst[(size_t)(q - dest * 2 * PP) * TX + line] = xq;
        }
    }
    if (CL > 1) cg::this_cluster().sync(); else __syncthreads();

    // ---------------- Stage C: back-substitution from shared memory ----------------------
    {
        const double *__restrict__ ta = s_a + (size_t)lp * m * TX + lx;
        const double *__restrict__ tc = s_c + (size_t)lp * m * TX + lx;
        const double *__restrict__ td = s_d + (size_t)lp * m * TX + lx;
        double *__restrict__ x = prm.x + off0;
        const double xf = yl[(size_t)(2 * lp) * TX + lx];
        const double xl = yl[(size_t)(2 * lp + 1) * TX + lx];
        st_stream(x, xf);
        st_stream(x + (size_t)(m - 1) * s, xl);
        double xn = xl;
#pragma unroll 4
        for (int r = m - 2; r >= 1; --r) {
            xn = fma(-tc[(size_t)r * TX], xn, fma(-ta[(size_t)r * TX], xf, td[(size_t)r * TX]));
            st_stream(x + r * s, xn);
        }
    }
}

// Pick TX / CL: TX = 32 lines (256 B row segments) when nx allows, then the smallest cluster that
// brings the per-CTA state under ~100 KB (two CTAs per SM, so that one CTA's load phase overlaps
// the other's reduced solve / back-substitution), else the smallest that fits at all.
inline bool configure_fused(FusedConfig *cfg, int nx, int ny, int P, int want_lines,
                            int want_cluster, const cudaDeviceProp &prop, const char **why)
{
    const int m = ny / P;
    const size_t max_smem = prop.sharedMemPerBlockOptin;
    const int tx_opts[4] = {32, 16, 8, 64};
    const int cl_opts[4] = {1, 2, 4, 8};
    FusedConfig best;
    for (int pass = 0; pass < 2 && best.lines == 0; ++pass) {
        const size_t limit = pass == 0 ? (size_t)100 * 1024 : max_smem;
        for (int ti = 0; ti < 4 && best.lines == 0; ++ti) {
            const int TX = tx_opts[ti];
            if (want_lines && TX != want_lines) continue;
            if (nx % TX) continue;
            for (int ci = 0; ci < 4; ++ci) {
                const int CL = cl_opts[ci];
                if (want_cluster && CL != want_cluster) continue;
                if (P % CL || TX % CL) continue;
                const int PP = P / CL, TXS = TX / CL;
                const int threads = TX * PP;
                if (threads > 1024 || threads < TXS) continue;
                const size_t smem = fused_smem_doubles(TX, PP, m, P, TXS) * sizeof(double);
                if (smem > limit) continue;
                best.lines = TX; best.cluster = CL; best.pp = PP; best.threads = threads;
                best.lines_solved = TXS; best.smem = smem;
                break;
            }
        }
    }
    if (best.lines == 0) {
        *why = "no (lines, cluster) choice fits shared memory / divisibility (nx % 8, P % cluster)";
        return false;
    }
    *cfg = best;
    return true;
}

template <int CL, int MAXT, int U>
inline cudaError_t launch_fused_inst(const FusedConfig &cfg, const FusedParams &prm, cudaStream_t st)
{
    cudaError_t e = cudaFuncSetAttribute(fused_kernel<CL, MAXT, U>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cfg.smem);
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t lc = {};
    lc.gridDim = dim3((unsigned)((size_t)prm.xtiles * prm.nzs * CL));
    lc.blockDim = dim3(cfg.threads);
    lc.dynamicSmemBytes = cfg.smem;
    lc.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CL; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    lc.attrs = attr;
    lc.numAttrs = CL > 1 ? 1 : 0;
    return cudaLaunchKernelEx(&lc, fused_kernel<CL, MAXT, U>, prm);
}

template <int CL>
inline cudaError_t launch_fused_cl(const FusedConfig &cfg, const FusedParams &prm, cudaStream_t st)
{
    if (cfg.threads <= 128) return launch_fused_inst<CL, 128, 8>(cfg, prm, st);
    if (cfg.threads <= 512) return launch_fused_inst<CL, 512, 4>(cfg, prm, st);
    return launch_fused_inst<CL, 1024, 2>(cfg, prm, st);
}

inline cudaError_t launch_fused(const FusedConfig &cfg, const double *a, const double *b,
                                const double *c, const double *d, double *x, int nx, int ny,
                                int nzs, int P, cudaStream_t st)
{
    FusedParams prm;
    prm.a = a; prm.b = b; prm.c = c; prm.d = d; prm.x = x;
    prm.nx = nx; prm.ny = ny; prm.nzs = nzs; prm.P = P; prm.m = ny / P;
    prm.TX = cfg.lines; prm.PP = cfg.pp; prm.TXS = cfg.lines_solved;
    prm.xtiles = nx / cfg.lines;
    switch (cfg.cluster) {
    case 1: return launch_fused_cl<1>(cfg, prm, st);
    case 2: return launch_fused_cl<2>(cfg, prm, st);
    case 4: return launch_fused_cl<4>(cfg, prm, st);
    case 8: return launch_fused_cl<8>(cfg, prm, st);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace tdma
