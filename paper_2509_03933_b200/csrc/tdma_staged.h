// STAGED variant (north_star: "shared-memory or TMA staging of short partition
// segments so the modified coefficients stay on chip instead of round-tripping HBM"): host-side
// interface between the plan (tdma_plan.cu) and the kernels' translation unit (tdma_staged.cu).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>

namespace tdma {

struct StagedConfig {
    int lines = 0, rows = 0, blocks_per_line = 0, leaf_rows = 0, leaves = 0, threads = 0, slots = 0;
    int lp = 0;         // tree levels run inside a CTA
    int lp_shift = 0;   // log2(leaves per exchanged node)
    int Pe = 0;         // partitions whose boundary equations are exchanged = rows / 2 of the reduced system
    size_t smem = 0;
    void *impl = nullptr;   // the TMA tiling (owned by the translation unit)
};

bool configure_staged(StagedConfig *out, int nx, int ny, int P, bool axis_z, const cudaDeviceProp &prop, const char **why);
void free_staged(StagedConfig *cfg);

// stage = 1 (A: reduce, writes ra / rc / rd [2 Pe][Lb]) or 2 (C: re-reduce + back-substitute, reads y).
// a, b, c, d, x: slice 0 of the batch; Lb = nx * nzs lines.  periodic: cyclic lines -- a_0 and c_{n-1} are
// kept, so rows 0 and 2 Pe - 1 of the reduced system couple each other (stage_b_cyclic_kernel).
cudaError_t launch_staged(StagedConfig &cfg, int stage, const double *a, const double *b, const double *c,
                          const double *d, double *x, double *ra, double *rc, double *rd, const double *y,
                          int nx, int ny, int nzs, long long rs, long long os, bool axis_z, cudaStream_t st,
                          bool periodic = false);

// y-slab decomposition (tdma_slab.cu): the launch holds rows row0 .. row0 + ny - 1 of lines of ny_total
// rows; stage 1 writes send[dest][Pe][6][Ls], stage 2 reads yrecv[src][2 Pe][Ls] (Ls = nx * nzs / ranks).
cudaError_t launch_staged_slab(StagedConfig &cfg, int stage, const double *a, const double *b, const double *c,
                               const double *d, double *x, double *send, const double *yrecv, int nx, int ny,
                               int nzs, int row0, int ny_total, long long Ls, cudaStream_t st,
                               double *const *peer = nullptr, long long peer_off = 0);

}  // namespace tdma
