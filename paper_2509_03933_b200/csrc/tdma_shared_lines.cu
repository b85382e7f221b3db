// Shared-coefficient / complex-RHS solve, the GENERAL-SHAPE kernel:
// one thread per line, plain Thomas over the whole line with the matrix rebuilt from the
// 1-D arrays on the fly.  It takes what the tiled TMA kernel (tdma_shared_tma.cuh) cannot: line lengths
// without a CL x 2^k x {4, 8, 16, 32} tiling, odd nx with real cells, complex cells along x, d / x that
// are only 8-byte aligned.  Not a fast path: c' travels through a plan-owned scratch array and d' through
// x, 48 bytes per real cell instead of 16; the lanes of a warp are consecutive lines, so y and z sweeps are
// coalesced and x sweeps are strided.
//
// Cyclic lines (options.periodic) by condensation on the last unknown, as in stage_b_cyclic_kernel:
// rows 0 .. n-2 form a plain system T with x_{n-1} as a parameter,  T x = d - x_{n-1} h0,
// h0 = a_0 e_0 + c_{n-2} e_{n-2};  one elimination of T carries d (g) and h0 (h),
//     x_{n-1} = (d_{n-1} - a_{n-1} g_{n-2} - c_{n-1} g_0) / (b_{n-1} - a_{n-1} h_{n-2} - c_{n-1} h_0),
//     x_j = g_j - h_j x_{n-1}.
#include "tdma_shared.h"

namespace tdma {

namespace {

// cell (lane i, row r, slice k) of d / x sits at  (k os + i ls + r rs) NC  doubles
template <int NC, bool kCyclic>
__global__ void __launch_bounds__(128) shared_lines_kernel(const SharedLineArgs p)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long L = (long long)p.lanes * p.slices;
    if (t >= L) return;
    const int k = (int)(t / p.lanes), i = (int)(t - (long long)k * p.lanes);
    const double s = (p.sx ? p.sx[i] : 0.0) + (p.sz ? p.sz[p.k0 + k] : 0.0);   // summed first (D4)
    const bool pin = p.pin00 && i == 0 && p.k0 + k == 0;
    const size_t base = ((size_t)k * (size_t)p.os + (size_t)i * (size_t)p.ls) * NC, rs = (size_t)p.rs * NC;
    const double *__restrict__ a = p.a_y, *__restrict__ b0 = p.b0_y, *__restrict__ c = p.c_y;
    const double *d = p.d + base;
    double *x = p.x + base;
    double *cs = p.cs + t, *hs = kCyclic ? p.hs + t : nullptr;      // [row][line], line fastest
    const size_t LL = (size_t)L;
    const int n = p.n, nt = kCyclic ? n - 1 : n;                    // rows of the plain system swept below

    // Rows are handled U at a time with the next U rows' loads issued first (the recurrences are serial
    // per thread; bandwidth comes from loads kept in flight, as in the stage kernels).  x may alias d
    // exactly: a row of d is always loaded before that row of x is stored.
    constexpr int U = 8;

    // forward elimination of rows 0 .. nt-1: c' -> cs, d' (g') -> x, h' -> hs
    double inv = 1.0 / (pin ? 1.0 : b0[0] - s);
    double cp = pin ? 0.0 : c[0] * inv, dp[NC], hp = 0.0;
#pragma unroll
    for (int q = 0; q < NC; ++q) dp[q] = d[q] * inv;
    if (kCyclic) hp = (a[0] + (nt == 1 ? c[0] : 0.0)) * inv;       // n = 2: both neighbours of x_0 are x_1
    double nd[U][NC];
#pragma unroll
    for (int u = 0; u < U; ++u)
        if (1 + u < nt) {
#pragma unroll
            for (int q = 0; q < NC; ++q) nd[u][q] = d[(size_t)(1 + u) * rs + q];
        }
#pragma unroll
    for (int q = 0; q < NC; ++q) x[q] = dp[q];
    cs[0] = cp;
    if (kCyclic) hs[0] = hp;
    for (int j0 = 1; j0 < nt; j0 += U) {
        double cd[U][NC];
#pragma unroll
        for (int u = 0; u < U; ++u) {
#pragma unroll
            for (int q = 0; q < NC; ++q) cd[u][q] = nd[u][q];
        }
#pragma unroll
        for (int u = 0; u < U; ++u)
            if (j0 + U + u < nt) {
#pragma unroll
                for (int q = 0; q < NC; ++q) nd[u][q] = d[(size_t)(j0 + U + u) * rs + q];
            }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int j = j0 + u;
            if (j < nt) {
                const double aj = a[j];
                inv = 1.0 / fma(-aj, cp, b0[j] - s);
#pragma unroll
                for (int q = 0; q < NC; ++q) {
                    dp[q] = fma(-aj, dp[q], cd[u][q]) * inv;
                    x[(size_t)j * rs + q] = dp[q];
                }
                if (kCyclic) { hp = fma(-aj, hp, j == nt - 1 ? c[j] : 0.0) * inv; hs[(size_t)j * LL] = hp; }
                cp = c[j] * inv;
                cs[(size_t)j * LL] = cp;
            }
        }
    }
    // back substitution of rows nt-2 .. 0 (row nt-1 is final already)
    double xv[NC], hv = hp, g_last[NC];
    const double h_last = hp;
#pragma unroll
    for (int q = 0; q < NC; ++q) xv[q] = g_last[q] = dp[q];
    double nc_[U], nh[U], nx_[U][NC];
#pragma unroll
    for (int u = 0; u < U; ++u) {
        const int j = nt - 2 - u;
        if (j >= 0) {
            nc_[u] = cs[(size_t)j * LL];
            if (kCyclic) nh[u] = hs[(size_t)j * LL];
#pragma unroll
            for (int q = 0; q < NC; ++q) nx_[u][q] = x[(size_t)j * rs + q];
        }
    }
    for (int j0 = nt - 2; j0 >= 0; j0 -= U) {
        double cc[U], ch[U], cx[U][NC];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            cc[u] = nc_[u]; ch[u] = nh[u];
#pragma unroll
            for (int q = 0; q < NC; ++q) cx[u][q] = nx_[u][q];
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int j = j0 - U - u;
            if (j >= 0) {
                nc_[u] = cs[(size_t)j * LL];
                if (kCyclic) nh[u] = hs[(size_t)j * LL];
#pragma unroll
                for (int q = 0; q < NC; ++q) nx_[u][q] = x[(size_t)j * rs + q];
            }
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int j = j0 - u;
            if (j >= 0) {
#pragma unroll
                for (int q = 0; q < NC; ++q) {
                    xv[q] = fma(-cc[u], xv[q], cx[u][q]);
                    x[(size_t)j * rs + q] = xv[q];
                }
                if (kCyclic) { hv = fma(-cc[u], hv, ch[u]); hs[(size_t)j * LL] = hv; }
            }
        }
    }
    if (!kCyclic) return;
    // xv, hv: row 0.  Row n-1 closes the ring.
    const int l = n - 1;
    const double den = 1.0 / fma(-c[l], hv, fma(-a[l], h_last, b0[l] - s));
    double xl[NC];
#pragma unroll
    for (int q = 0; q < NC; ++q) {
        xl[q] = fma(-c[l], xv[q], fma(-a[l], g_last[q], d[(size_t)l * rs + q])) * den;
        x[(size_t)l * rs + q] = xl[q];
    }
    for (int j0 = 0; j0 < nt; j0 += U) {
        double ch[U], cx[U][NC];
#pragma unroll
        for (int u = 0; u < U; ++u)
            if (j0 + u < nt) {
                ch[u] = hs[(size_t)(j0 + u) * LL];
#pragma unroll
                for (int q = 0; q < NC; ++q) cx[u][q] = x[(size_t)(j0 + u) * rs + q];
            }
#pragma unroll
        for (int u = 0; u < U; ++u)
            if (j0 + u < nt) {
#pragma unroll
                for (int q = 0; q < NC; ++q) x[(size_t)(j0 + u) * rs + q] = fma(-ch[u], xl[q], cx[u][q]);
            }
    }
}

}  // namespace

cudaError_t launch_shared_lines(const SharedLineArgs &p, cudaStream_t st)
{
    const long long L = (long long)p.lanes * p.slices;
    if (L <= 0) return cudaSuccess;
    const unsigned grid = (unsigned)((L + 127) / 128);
    if (p.ncomp == 2) {
        if (p.periodic) shared_lines_kernel<2, true><<<grid, 128, 0, st>>>(p);
        else shared_lines_kernel<2, false><<<grid, 128, 0, st>>>(p);
    } else {
        if (p.periodic) shared_lines_kernel<1, true><<<grid, 128, 0, st>>>(p);
        else shared_lines_kernel<1, false><<<grid, 128, 0, st>>>(p);
    }
    return cudaGetLastError();
}

}  // namespace tdma
