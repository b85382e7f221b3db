// Stage kernels of the PIPELINED variant (sm_100a): partition reduce (stage A, with the gather
// fused as its epilogue or as a separate A2B kernel), reduced 2P-row solve (stage B) and
// back-substitution (stage C).  PAPER.md:49-58 (five stages), Alg. 2 PAPER.md:166-214.
//
// Thread mapping (all three): one thread per (line, partition) -- or per line for stage B -- with
// consecutive threads on consecutive x, so every row access of a warp is one 256 B segment.
// The recurrences along y are serial per thread; bandwidth comes from U rows x 3-4 arrays of
// independent loads kept in flight per thread (register double buffer).
//
// Arithmetic of one partition (local rows r = 0..m-1, x_{-1} = previous partition's last unknown,
// x_m = next partition's first; global a_0 := 0, c_{ny-1} := 0):
//   rows 0 and 1 are normalised by their b;
//   r = 2..m-1 (forward elimination with x_0 kept as a parameter):
//        inv = 1/(b_r - a_r c'_{r-1});  d'_r = (d_r - a_r d'_{r-1}) inv;  c'_r = c_r inv;
//        a'_r = -a_r a'_{r-1} inv          =>  a'_r x_0 + x_r + c'_r x_{r+1} = d'_r   (r >= 1)
//   while sweeping, row r-1 is folded into the FIRST-ROW equation
//        fa x_{-1} + fb x_0 + fc x_{r-1} = fd   ->   fb -= fc a'_{r-1}; fd -= fc d'_{r-1};
//        fc = -fc c'_{r-1}                      (now couples x_r)
//   so that after the sweep it reads fa x_{-1} + fb x_0 + fc x_{m-1} = fd and is normalised by fb.
//   Reduced rows (unit diagonal): 2p = (fa, fc | fd)/fb, 2p+1 = (a'_{m-1}, c'_{m-1} | d'_{m-1}).
//   Stage C: x_0 = Y[2p], x_{m-1} = Y[2p+1], r = m-2..1: x_r = d'_r - a'_r x_0 - c'_r x_{r+1}.
// One division per cell; nothing is re-read inside stage A.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tdma {

// read-once inputs / write-once output: streaming (evict-first) so they do not displace the
// scratch ring in L2; scratch and reduced buffers: L2-only (.cg), they are re-read by the next stage
__device__ __forceinline__ double ld_stream(const double *p) { return __ldcs(p); }
__device__ __forceinline__ void st_stream(double *p, double v) { __stcs(p, v); }
__device__ __forceinline__ double ld_keep(const double *p) { return __ldcg(p); }
__device__ __forceinline__ void st_keep(double *p, double v) { __stcg(p, v); }

struct StageParams {
    const double *a, *b, *c, *d;  // batch base (slice k0 of the slab)
    double *x;                    // batch base of the output
    double *sa, *sc, *sd;         // scratch slot, batch layout [bz][ny][nx]
    double *ra, *rc, *rd, *cp, *y;  // reduced system [2P][Lb], line fastest
    double *send;                 // separate gather: send_A buffer [P][6][Lb]
    long long Lb;                 // lines in this batch = nx * slices
    int nx, ny, m, P;             // ny = rows per line (the solve axis), slices = the other axis
    long long rs, os;             // caller arrays: element stride between rows of a line / between
                                  // slices (y sweep: nx, nx*ny; z sweep: nx*ny, nx); scratch is
                                  // always [slice][row][x]
    long long ls = 1;             // ... and between neighbouring lines of a slice: 1, except for x sweeps
                                  // (lines along the contiguous axis: rs = 1, ls = line length; the
                                  // accesses of a warp are then strided -- the fallback for x sweeps
                                  // the TMA kernel cannot tile)
    // y-slab decomposition (tdma_slab.cu): this launch holds partitions pg0 .. pg0+P-1
    // of Ptot; the lines of a batch are dealt out evenly, Ls to each rank (single GPU: 0, P, 0)
    int pg0 = 0, Ptot = 0;
    long long Ls = 0;
    // peer stores (tdma_slab_stage_a_peer / _b_peer): the block of the send / yout buffer meant for
    // rank q is written straight into rank q's receive buffer, peer[q] + peer_off (device table of
    // nranks pointers; peer_off = this rank's block in the receiver's [src] layout); peer_rows =
    // rows of Ls doubles per block of yout (2 P_local)
    double *const *peer = nullptr;
    long long peer_off = 0;
    int peer_rows = 0;
    // cyclic lines (options.periodic): a_0 couples x_{n-1} and c_{n-1} couples x_0; stage A keeps both
    // entries, which makes the reduced system cyclic (stage_b_cyclic_kernel); stage C is unchanged
    int cyclic = 0;
};

// row q of stage B's solution for line l (slab: yout[dest][2 P_local][Ls], or the peer's yrecv block)
__device__ __forceinline__ double *y_row(const StageParams &prm, int q, long long l)
{
    if (prm.peer) {
        const int dest = q / prm.peer_rows;
        return prm.peer[dest] + (prm.peer_off + (long long)(q - dest * prm.peer_rows) * prm.Lb + l);
    }
    return prm.y + (size_t)q * (size_t)prm.Lb + l;
}

// where stage A's two boundary equations per (line, partition) go
enum { kOutReduced = 0,   // RA / RC / RD rows 2p, 2p+1 (gather fused into the epilogue)
       kOutSendA = 1,     // send_A[P][6][Lb] for the separate gather kernel
       kOutSlab = 2 };    // send[dest rank][P][6][Ls], dest = l / Ls: the all-to-all's send buffer

// ------------------------------------------------------------------------------------------
// Stage A
// ------------------------------------------------------------------------------------------
template <int U, int kOut>
__global__ void __launch_bounds__(128) stage_a_kernel(const StageParams prm)
{
    const long long l = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (l >= prm.Lb) return;
    const int p = blockIdx.y;
    const int nx = prm.nx, m = prm.m;
    const long long kk = l / nx;
    const int i = (int)(l - kk * nx);
    const size_t off0 = (size_t)kk * (size_t)prm.os + (size_t)i * (size_t)prm.ls + (size_t)p * m * (size_t)prm.rs;
    const size_t soff0 = (size_t)kk * (size_t)prm.ny * nx + i + (size_t)p * m * (size_t)nx;
    const double *__restrict__ a = prm.a + off0;
    const double *__restrict__ b = prm.b + off0;
    const double *__restrict__ c = prm.c + off0;
    const double *__restrict__ d = prm.d + off0;
    double *__restrict__ sa = prm.sa + soff0;
    double *__restrict__ sc = prm.sc + soff0;
    double *__restrict__ sd = prm.sd + soff0;
    const size_t s = (size_t)prm.rs, ss = (size_t)nx;
    const bool first_part = !prm.cyclic && (prm.pg0 + p == 0), last_part = !prm.cyclic && (prm.pg0 + p == prm.Ptot - 1);

    // first-row equation  fa x_{-1} + fb x_0 + fc x_frontier = fd
    double inv = 1.0 / ld_stream(b);
    double fa = first_part ? 0.0 : ld_stream(a) * inv;
    double fc = ld_stream(c) * inv;
    double fd = ld_stream(d) * inv;
    double fb = 1.0;
    // row 1 in forward form  pa x_0 + x_1 + pc x_2 = pd
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
        for (int u = 0; u < U; ++u) {                    // next chunk's loads go out first
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
                // fold row r-1 into the first-row equation, then hand it to stage C
                fb = fma(-fc, pa, fb);
                fd = fma(-fc, pd, fd);
                fc = -fc * pc;
                st_keep(sa + (r - 1) * ss, pa);
                st_keep(sc + (r - 1) * ss, pc);
                st_keep(sd + (r - 1) * ss, pd);
                const double ar = ca[u];
                const double cr = (last_part && r == m - 1) ? 0.0 : cc[u];
                inv = 1.0 / fma(-ar, pc, cb[u]);
                pd = fma(-ar, pd, cd[u]) * inv;
                pc = cr * inv;
                pa = -(ar * pa) * inv;
            }
        }
    }
    // m == 2: first-row equation is already (fa, 1, fc | fd) with frontier x_1 = x_{m-1}
    inv = 1.0 / fb;
    const size_t Lb = (size_t)prm.Lb;
    if (kOut == kOutSendA) {
        double *__restrict__ sp = prm.send + (size_t)p * 6 * Lb + l;
        st_keep(sp, fa * inv); st_keep(sp + Lb, fc * inv); st_keep(sp + 2 * Lb, fd * inv);
        st_keep(sp + 3 * Lb, pa); st_keep(sp + 4 * Lb, pc); st_keep(sp + 5 * Lb, pd);
    } else if (kOut == kOutSlab) {
        const size_t Ls = (size_t)prm.Ls, dest = (size_t)l / Ls, j = (size_t)l - dest * Ls;
        double *__restrict__ sp = prm.peer ? prm.peer[dest] + ((size_t)prm.peer_off + (size_t)p * 6 * Ls + j)
                                           : prm.send + ((dest * prm.P + p) * 6) * Ls + j;
        st_keep(sp, fa * inv); st_keep(sp + Ls, fc * inv); st_keep(sp + 2 * Ls, fd * inv);
        st_keep(sp + 3 * Ls, pa); st_keep(sp + 4 * Ls, pc); st_keep(sp + 5 * Ls, pd);
    } else {
        const size_t q0 = (size_t)(2 * p) * Lb + l, q1 = q0 + Lb;
        st_keep(prm.ra + q0, fa * inv); st_keep(prm.rc + q0, fc * inv); st_keep(prm.rd + q0, fd * inv);
        st_keep(prm.ra + q1, pa); st_keep(prm.rc + q1, pc); st_keep(prm.rd + q1, pd);
    }
}

// Separate A2B gather ("Save data in send_A" / "Get data from recv_B"):
// send[p][6][Lb] -> RA/RC/RD[2P][Lb].  One thread per (line, partition).
static __global__ void __launch_bounds__(256) gather_kernel(const StageParams prm)
{
    const long long l = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (l >= prm.Lb) return;
    const int p = blockIdx.y;
    const size_t Lb = (size_t)prm.Lb;
    const double *__restrict__ sp = prm.send + (size_t)p * 6 * Lb + l;
    const size_t q0 = (size_t)(2 * p) * Lb + l, q1 = q0 + Lb;
    st_keep(prm.ra + q0, ld_keep(sp)); st_keep(prm.rc + q0, ld_keep(sp + Lb));
    st_keep(prm.rd + q0, ld_keep(sp + 2 * Lb));
    st_keep(prm.ra + q1, ld_keep(sp + 3 * Lb)); st_keep(prm.rc + q1, ld_keep(sp + 4 * Lb));
    st_keep(prm.rd + q1, ld_keep(sp + 5 * Lb));
}

// ------------------------------------------------------------------------------------------
// Stage B: Thomas on the 2P-row reduced system (unit diagonal), one thread per line.
// Low occupancy by construction; runs on its own high-priority stream.
// ------------------------------------------------------------------------------------------
template <int U>
__global__ void __launch_bounds__(64) stage_b_kernel(const StageParams prm)
{
    const long long l = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (l >= prm.Lb) return;
    const size_t Lb = (size_t)prm.Lb;
    const int Q = 2 * prm.P;
    const double *__restrict__ ra = prm.ra + l;
    const double *__restrict__ rc = prm.rc + l;
    const double *rd = prm.rd + l;
    double *__restrict__ cpb = prm.cp + l;
    // the forward-eliminated right-hand side d' is parked in y; with peer stores y is remote memory
    // that is written once, and d' overwrites RD in place (row q is stored after it was loaded)
    double *tmp = prm.peer ? prm.rd + l : prm.y + l;

    double cp = ld_keep(rc), dp = ld_keep(rd);          // row 0: sub-diagonal is 0
    st_keep(cpb, cp); st_keep(tmp, dp);
    double na[U], nc[U], nd[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
        const int q = 1 + u;
        if (q < Q) { na[u] = ld_keep(ra + q * Lb); nc[u] = ld_keep(rc + q * Lb); nd[u] = ld_keep(rd + q * Lb); }
    }
    for (int q0 = 1; q0 < Q; q0 += U) {
        double ca[U], cc[U], cd[U];
#pragma unroll
        for (int u = 0; u < U; ++u) { ca[u] = na[u]; cc[u] = nc[u]; cd[u] = nd[u]; }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int q = q0 + U + u;
            if (q < Q) { na[u] = ld_keep(ra + q * Lb); nc[u] = ld_keep(rc + q * Lb); nd[u] = ld_keep(rd + q * Lb); }
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int q = q0 + u;
            if (q < Q) {
                const double inv = 1.0 / fma(-ca[u], cp, 1.0);
                dp = fma(-ca[u], dp, cd[u]) * inv;
                cp = cc[u] * inv;
                st_keep(cpb + q * Lb, cp);
                st_keep(tmp + q * Lb, dp);
            }
        }
    }
    // back substitution; the last row's cp is 0 by construction (c_{ny-1} := 0)
    double xq = dp;
    st_keep(y_row(prm, Q - 1, l), xq);
    for (int q = Q - 2; q >= 0; --q) {
        xq = fma(-ld_keep(cpb + q * Lb), xq, ld_keep(tmp + q * Lb));
        st_keep(y_row(prm, q, l), xq);
    }
}

// ------------------------------------------------------------------------------------------
// Stage B for CYCLIC lines (options.periodic; the periodic sweeps of BASELINE cfg 4).
// Stage A then leaves a_0 and c_{n-1} in place, so row 0 of the reduced system couples y_{Q-1}
// through ra_0 and row Q-1 couples y_0 through rc_{Q-1}: a cyclic tridiagonal system with unit
// diagonal -- the wrap is resolved here, at the level of the paper's reduced system, and nothing
// else changes (no Sherman-Morrison pass over the full lines).  Condensation on the last unknown:
// rows 0 .. Q-2 are a plain tridiagonal system T in y_0 .. y_{Q-2} with y_{Q-1} as a parameter,
//     T y = rd - y_{Q-1} h0 ,    h0 = ra_0 e_0 + rc_{Q-2} e_{Q-2} ,
// one forward elimination of T carries both right-hand sides (g' for rd, h' for h0), the back
// substitution gives y_i = g_i - h_i y_{Q-1}, and row Q-1 fixes
//     y_{Q-1} = (rd_{Q-1} - ra_{Q-1} g_{Q-2} - rc_{Q-1} g_0) / (1 - ra_{Q-1} h_{Q-2} - rc_{Q-1} h_0).
// h' / h overwrite RA in place (a row is stored after it was loaded), g' / g sit where stage B parks d'.
// ------------------------------------------------------------------------------------------
static __global__ void __launch_bounds__(64) stage_b_cyclic_kernel(const StageParams prm)
{
    const long long l = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (l >= prm.Lb) return;
    const size_t Lb = (size_t)prm.Lb;
    const int Q = 2 * prm.P, n = Q - 1;                  // T has n >= 1 rows
    double *ra = prm.ra + l;
    const double *__restrict__ rc = prm.rc + l;
    const double *rd = prm.rd + l;
    double *__restrict__ cpb = prm.cp + l;
    double *tmp = prm.peer ? prm.rd + l : prm.y + l;

    double cp = ld_keep(rc), gp = ld_keep(rd), hp = ld_keep(ra);
    if (n == 1) hp += cp;                                // Q = 2: both neighbours of y_0 are y_1
    st_keep(cpb, cp); st_keep(tmp, gp); st_keep(ra, hp);
    for (int q = 1; q < n; ++q) {
        const double aq = ld_keep(ra + q * Lb), cq = ld_keep(rc + q * Lb), dq = ld_keep(rd + q * Lb);
        const double inv = 1.0 / fma(-aq, cp, 1.0);
        gp = fma(-aq, gp, dq) * inv;
        hp = fma(-aq, hp, q == n - 1 ? cq : 0.0) * inv;
        cp = cq * inv;
        st_keep(cpb + q * Lb, cp); st_keep(tmp + q * Lb, gp); st_keep(ra + q * Lb, hp);
    }
    double g = gp, h = hp;                               // row n-1 of T
    const double g_last = g, h_last = h;
    for (int q = n - 2; q >= 0; --q) {
        const double cq = ld_keep(cpb + q * Lb);
        g = fma(-cq, g, ld_keep(tmp + q * Lb));
        h = fma(-cq, h, ld_keep(ra + q * Lb));
        st_keep(tmp + q * Lb, g); st_keep(ra + q * Lb, h);
    }
    // g, h: row 0.  Row Q-1 of the reduced system was not touched above.
    const double aL = ld_keep(ra + (size_t)n * Lb), cL = ld_keep(rc + (size_t)n * Lb), dL = ld_keep(rd + (size_t)n * Lb);
    const double yl = fma(-cL, g, fma(-aL, g_last, dL)) / fma(-cL, h, fma(-aL, h_last, 1.0));
    st_keep(y_row(prm, Q - 1, l), yl);
    for (int q = 0; q < n; ++q)
        st_keep(y_row(prm, q, l), fma(-ld_keep(ra + q * Lb), yl, ld_keep(tmp + q * Lb)));
}

// ------------------------------------------------------------------------------------------
// Stage B, PDD variant (Sun 1995): no chain over the 2P rows.  The reduced rows
//      fa y_l(p-1) + x_f + fc x_l = fd ,      pa x_f + x_l + pc y_f(p+1) = pd
// of partition p are first solved for (x_f, x_l) as functions of the NEIGHBOURS' interface
// unknowns (the partition's own 2 x 2 block, det = 1 - fc pa):
//      x_f = xt0 - v0 y_l(p-1) - w0 y_f(p+1) ,   x_l = xtl - vl y_l(p-1) - wl y_f(p+1)
// -- xt, v, w are the first / last entries of Sun's block solution and spikes.  PDD drops the far
// spike ends w0 and vl, which leaves one 2 x 2 system per interface,
//      y_l(p) + wl(p) y_f(p+1) = xtl(p) ,     v0(p+1) y_l(p) + y_f(p+1) = xt0(p+1) ,
// and then evaluates x_f, x_l with all four spike ends.  One thread per (line, partition): it
// rebuilds the spike ends of its two neighbours from their rows (18 coalesced loads, no
// dependence on any other thread).  Exact when partitions do not couple; error of the order of
// the dropped entries otherwise (strictly dominant systems: geometric in ny/P).
// ------------------------------------------------------------------------------------------
struct SpikeEnds { double xt0, v0, w0, xtl, vl, wl; };

__device__ __forceinline__ SpikeEnds spike_ends(const double *__restrict__ ra, const double *__restrict__ rc,
                                                const double *__restrict__ rd, size_t q0, size_t Lb)
{
    const double fa = ld_keep(ra + q0), fc = ld_keep(rc + q0), fd = ld_keep(rd + q0);
    const double pa = ld_keep(ra + q0 + Lb), pc = ld_keep(rc + q0 + Lb), pd = ld_keep(rd + q0 + Lb);
    const double inv = 1.0 / fma(-fc, pa, 1.0);
    SpikeEnds s;
    s.xt0 = fma(-fc, pd, fd) * inv; s.v0 = fa * inv; s.w0 = -(fc * pc) * inv;
    s.xtl = fma(-pa, fd, pd) * inv; s.vl = -(pa * fa) * inv; s.wl = pc * inv;
    return s;
}

static __global__ void __launch_bounds__(128) stage_b_pdd_kernel(const StageParams prm)
{
    const long long l = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (l >= prm.Lb) return;
    const int p = blockIdx.y, P = prm.P;
    const size_t Lb = (size_t)prm.Lb;
    const SpikeEnds me = spike_ends(prm.ra, prm.rc, prm.rd, (size_t)(2 * p) * Lb + l, Lb);
    double y_prev = 0.0, y_next = 0.0;        // y_l(p-1), y_f(p+1)
    if (p > 0) {
        const SpikeEnds lo = spike_ends(prm.ra, prm.rc, prm.rd, (size_t)(2 * p - 2) * Lb + l, Lb);
        y_prev = fma(-lo.wl, me.xt0, lo.xtl) / fma(-lo.wl, me.v0, 1.0);
    }
    if (p < P - 1) {
        const SpikeEnds hi = spike_ends(prm.ra, prm.rc, prm.rd, (size_t)(2 * p + 2) * Lb + l, Lb);
        y_next = fma(-hi.v0, me.xtl, hi.xt0) / fma(-me.wl, hi.v0, 1.0);
    }
    st_keep(y_row(prm, 2 * p, l), fma(-me.w0, y_next, fma(-me.v0, y_prev, me.xt0)));
    st_keep(y_row(prm, 2 * p + 1, l), fma(-me.wl, y_next, fma(-me.vl, y_prev, me.xtl)));
}

// ------------------------------------------------------------------------------------------
// Stage C: back-substitution inside each partition, one thread per (line, partition).
// ------------------------------------------------------------------------------------------
// kSlab: x_first / x_last come from the all-to-all's receive buffer yrecv[src rank][2 P][Ls] (prm.y),
// src = l / Ls (the rank that solved the line's reduced system).
template <int U, bool kSlab = false>
__global__ void __launch_bounds__(128) stage_c_kernel(const StageParams prm)
{
    const long long l = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (l >= prm.Lb) return;
    const int p = blockIdx.y;
    const int nx = prm.nx, m = prm.m;
    const long long kk = l / nx;
    const int i = (int)(l - kk * nx);
    const size_t off0 = (size_t)kk * (size_t)prm.os + (size_t)i * (size_t)prm.ls + (size_t)p * m * (size_t)prm.rs;
    const size_t soff0 = (size_t)kk * (size_t)prm.ny * nx + i + (size_t)p * m * (size_t)nx;
    const double *__restrict__ sa = prm.sa + soff0;
    const double *__restrict__ sc = prm.sc + soff0;
    const double *__restrict__ sd = prm.sd + soff0;
    double *__restrict__ x = prm.x + off0;
    const size_t s = (size_t)prm.rs, ss = (size_t)nx;
    const size_t Lb = (size_t)prm.Lb;

    double xf, xl;
    if (kSlab) {
        const size_t Ls = (size_t)prm.Ls, src = (size_t)l / Ls, j = (size_t)l - src * Ls;
        const double *__restrict__ yp = prm.y + (src * 2 * prm.P + 2 * p) * Ls + j;
        xf = ld_keep(yp); xl = ld_keep(yp + Ls);
    } else {
        xf = ld_keep(prm.y + (size_t)(2 * p) * Lb + l);
        xl = ld_keep(prm.y + (size_t)(2 * p + 1) * Lb + l);
    }
    st_stream(x, xf);
    st_stream(x + (size_t)(m - 1) * s, xl);
    double xn = xl;

    double na[U], nc[U], nd[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
        const int r = m - 2 - u;
        if (r >= 1) { na[u] = ld_keep(sa + r * ss); nc[u] = ld_keep(sc + r * ss); nd[u] = ld_keep(sd + r * ss); }
    }
    for (int r0 = m - 2; r0 >= 1; r0 -= U) {
        double ca[U], cc[U], cd[U];
#pragma unroll
        for (int u = 0; u < U; ++u) { ca[u] = na[u]; cc[u] = nc[u]; cd[u] = nd[u]; }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int r = r0 - U - u;
            if (r >= 1) { na[u] = ld_keep(sa + r * ss); nc[u] = ld_keep(sc + r * ss); nd[u] = ld_keep(sd + r * ss); }
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int r = r0 - u;
            if (r >= 1) {
                xn = fma(-cc[u], xn, fma(-ca[u], xf, cd[u]));
                st_stream(x + r * s, xn);
            }
        }
    }
}

// ny == 1 (only possible with P == 1): x = d / b.
static __global__ void __launch_bounds__(256) diagonal_kernel(const double *__restrict__ b,
                                                       const double *__restrict__ d,
                                                       double *__restrict__ x, size_t n)
{
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t < n) x[t] = d[t] / b[t];
}

}  // namespace tdma
