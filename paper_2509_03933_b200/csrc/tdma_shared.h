// Shared-coefficient / complex-RHS mode: host-side interface between the plan
// (tdma_plan.cu) and the kernel's translation unit (tdma_shared.cu).  Plain C++, no kernels here.
//
// The paper's own workload: complex-valued fields, a coefficient matrix that
// "depends solely on grid spacing" and the FFT-reduced Poisson operator
// (d2/dy2 - k_l - k_m): line (i,k) has a_j = a_y[j], c_j = c_y[j],
// b_j = b0_y[j] - (sx[i] + sz[k]); d and x carry ncomp = 1 (real) or 2 (complex, interleaved
// re/im) right-hand sides per cell.  HBM traffic: 8 ncomp bytes read + 8 ncomp written per cell.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>

namespace tdma {

struct SharedConfig {
    int ncomp = 0;      // NC: right-hand sides per cell
    int lines = 0;      // TX: lines (cells along x) per tile
    int cluster = 0;    // CL
    int rows = 0;       // R = ny / CL
    int leaf_rows = 0;  // M0
    int leaves = 0;     // W = R / M0 (power of two, <= 32)
    int threads = 0;    // W * TX
    int box_rows = 0;   // rows per TMA box (<= 256), divides R
    int slots = 0;      // NA: ring slots of one d / x tile each (>= 2)
    int uniform = 0;    // uniform matrix (no shift arrays): matrix work hoisted out of the tile loop
    int xsweep = 0;     // lines along the contiguous axis: 4-D tensor map, [leaf][line][16 x] slots
    int ctas_per_sm = 1;   // 2: the <= 128-register instantiation, two CTAs share an SM
    int max_clusters = 0;  // co-resident clusters (persistent grid), filled at first launch
    size_t smem = 0;
};

struct SharedArgs {
    const double *a_y, *b0_y, *c_y;   // [ny]   device
    const double *sx, *sz;            // [nx], [nz] device; sz already offset to slice 0 of the launch
    const double *d;                  // slice 0 of the launch
    double *x;
    int pin00;                        // row 0 of line (0, 0) of THIS launch's slice 0 is b = 1, c = 0
    int nx, ny, nzs;                  // lanes, rows per line, slices of the launch
    long long rs = 0, os = 0;         // cells between rows of a line / between slices of d and x
    int uniform = 0;                  // sx = sz = NULL: the same matrix for every line (needs SharedConfig::uniform)
    int axis_z = 0, periodic = 0;     // z sweep (rows are the slow axis); cyclic lines
                                      // x sweep: SharedConfig::xsweep; nx = lanes (caller's ny), ny = rows (caller's nx)
};

// Tiling for ny-row lines: CL x W x M0 with W a power of two.  want_* = 0: auto.
bool configure_shared(SharedConfig *out, int nx, int ny, int ncomp, int want_lines, int want_cluster,
                      int want_leaf, int want_slots, int want_ctas, const cudaDeviceProp &prop, const char **why,
                      bool xsweep = false, bool uniform = false);

// nzs = 0: prepare only (function attributes, persistent grid size).
cudaError_t launch_shared(SharedConfig &cfg, const SharedArgs &args, cudaStream_t st);

// General-shape kernel (tdma_shared_lines.cu): one thread per line, plain Thomas over the whole line.
struct SharedLineArgs {
    const double *a_y, *b0_y, *c_y;   // [n] device
    const double *sx, *sz;            // [lanes], [all slices] device, or both NULL (uniform matrix)
    const double *d;                  // slice k0
    double *x;
    double *cs, *hs;                  // scratch [n][lanes * slices] each; hs for cyclic lines only
    int n, lanes, slices, k0;         // rows per line, lines side by side, slices of this launch, its first slice
    long long rs, ls, os;             // CELLS between rows of a line / neighbouring lines / slices
    int ncomp, pin00, periodic;
};
cudaError_t launch_shared_lines(const SharedLineArgs &args, cudaStream_t st);

}  // namespace tdma
