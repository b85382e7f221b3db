// Translation unit of the STAGED variant's kernels: fused_tma_kernel with kStage = 1 (stage A) and
// kStage = 2 (stage C), independent CTAs, y / z sweeps of plain lines.
#include "tdma_fused_tma.cuh"
#include "tdma_staged.h"

namespace tdma {

bool configure_staged(StagedConfig *out, int nx, int ny, int P, bool axis_z, const cudaDeviceProp &prop, const char **why)
{
    if (!get_encode_tiled()) { *why = "cuTensorMapEncodeTiled not found"; return false; }
    TmaFusedConfig *t = new TmaFusedConfig[2];   // one per stage kernel: attributes and grid size are set per kernel
    if (!configure_tma_fused(t, nx, ny, P, 0, 0, 0, prop, why, false, axis_z, 0)) { delete[] t; return false; }
    if (t->threads > 256) {
        *why = "staged kernels are built for <= 256 threads per CTA";
        delete[] t;
        return false;
    }
    // exchanged level: the highest tree level whose nodes are no longer than a partition of the
    // paper (ny / P rows); leaves longer than a partition are exchanged as they are (D1)
    const int m = ny / P;
    int lp = 0, shift = 0;
    for (int nodes = t->leaves; nodes > 1;) {
        const int lkb = (nodes & 3) == 0 ? 2 : 1;
        if ((long)t->leaf_rows << (shift + lkb) > (long)m) break;
        shift += lkb; nodes >>= lkb; ++lp;
    }
    out->lines = t->lines; out->rows = t->rows; out->blocks_per_line = t->cluster; out->leaf_rows = t->leaf_rows;
    out->leaves = t->leaves; out->threads = t->threads; out->slots = t->slots; out->smem = t->smem;
    out->lp = lp; out->lp_shift = shift;
    out->Pe = ny / (t->leaf_rows << shift);
    t[1] = t[0];
    out->impl = t;
    return true;
}

void free_staged(StagedConfig *cfg)
{
    delete[] static_cast<TmaFusedConfig *>(cfg->impl);
    cfg->impl = nullptr;
}

template <int TX, int kStage>
static cudaError_t launch_staged_tx(TmaFusedConfig &t, const CUtensorMap *tm, const TmaFusedParams &prm, cudaStream_t st)
{
    switch (t.leaf_rows) {
    case 16: return launch_tma_inst<TX, 16, false, 256, false, kStage>(t, tm, prm, st);
    case 12: return launch_tma_inst<TX, 12, false, 256, false, kStage>(t, tm, prm, st);
    case 10: return launch_tma_inst<TX, 10, false, 256, false, kStage>(t, tm, prm, st);
    case 8: return launch_tma_inst<TX, 8, false, 256, false, kStage>(t, tm, prm, st);
    case 6: return launch_tma_inst<TX, 6, false, 256, false, kStage>(t, tm, prm, st);
    case 4: return launch_tma_inst<TX, 4, false, 256, false, kStage>(t, tm, prm, st);
    case 2: return launch_tma_inst<TX, 2, false, 256, false, kStage>(t, tm, prm, st);
    default: return cudaErrorInvalidValue;
    }
}

static cudaError_t launch_staged_any(StagedConfig &cfg, int stage, const double *a, const double *b, const double *c,
                                     const double *d, double *x, double *ra, double *rc, double *rd, const double *y,
                                     int nx, int ny, int nzs, long long rs, long long os, bool axis_z, int row0,
                                     int ny_total, long long Ls, double *const *peer, long long peer_off, cudaStream_t st,
                                     bool periodic = false)
{
    if (stage != 1 && stage != 2) return cudaErrorInvalidValue;
    TmaFusedConfig &t = static_cast<TmaFusedConfig *>(cfg.impl)[stage - 1];
    CUtensorMap tm[5];
    const void *ptr[5] = {a, b, c, d, x ? (const void *)x : (const void *)d};   // stage A never touches x
    for (int i = 0; i < 5 && nzs > 0; ++i)
        if (!make_slab_tensor_map(&tm[i], ptr[i], nx, ny, nzs, rs, os, axis_z, t.lines, t.box_rows)) return cudaErrorInvalidValue;
    TmaFusedParams prm;
    prm.nx = nx; prm.ny = ny; prm.nzs = nzs;
    prm.x = x;
    prm.rs = rs; prm.os = os; prm.axis_z = axis_z ? 1 : 0; prm.periodic = periodic ? 1 : 0;
    prm.CL = t.cluster; prm.R = t.rows; prm.W = t.leaves; prm.NS = t.slots;
    prm.xtiles = (nx + t.lines - 1) / t.lines;
    prm.ntiles = prm.xtiles * nzs;
    prm.box_rows = t.box_rows; prm.nbox = t.rows / t.box_rows;
    prm.red_a = ra; prm.red_c = rc; prm.red_d = rd; prm.red_y = y;
    prm.Lb = (long long)nx * nzs;
    prm.lp = cfg.lp; prm.lp_shift = cfg.lp_shift;
    prm.row0 = row0; prm.ny_total = ny_total; prm.Ls = Ls; prm.Pl = cfg.Pe;
    prm.red_peer = peer; prm.red_peer_off = peer_off;
    cudaError_t e;
    if (stage == 1) {
        switch (t.lines) {
        case 32: e = launch_staged_tx<32, 1>(t, tm, prm, st); break;
        case 16: e = launch_staged_tx<16, 1>(t, tm, prm, st); break;
        case 8: e = launch_staged_tx<8, 1>(t, tm, prm, st); break;
        default: e = cudaErrorInvalidValue;
        }
    } else {
        switch (t.lines) {
        case 32: e = launch_staged_tx<32, 2>(t, tm, prm, st); break;
        case 16: e = launch_staged_tx<16, 2>(t, tm, prm, st); break;
        case 8: e = launch_staged_tx<8, 2>(t, tm, prm, st); break;
        default: e = cudaErrorInvalidValue;
        }
    }
    return e;
}

cudaError_t launch_staged(StagedConfig &cfg, int stage, const double *a, const double *b, const double *c,
                          const double *d, double *x, double *ra, double *rc, double *rd, const double *y,
                          int nx, int ny, int nzs, long long rs, long long os, bool axis_z, cudaStream_t st,
                          bool periodic)
{
    return launch_staged_any(cfg, stage, a, b, c, d, x, ra, rc, rd, y, nx, ny, nzs, rs, os, axis_z, 0, 0, 0, nullptr, 0, st,
                             periodic);
}

cudaError_t launch_staged_slab(StagedConfig &cfg, int stage, const double *a, const double *b, const double *c,
                               const double *d, double *x, double *send, const double *yrecv, int nx, int ny,
                               int nzs, int row0, int ny_total, long long Ls, cudaStream_t st, double *const *peer,
                               long long peer_off)
{
    return launch_staged_any(cfg, stage, a, b, c, d, x, send, nullptr, nullptr, yrecv, nx, ny, nzs, (long long)nx,
                             (long long)nx * ny, false, row0, ny_total, Ls, peer, peer_off, st);
}

}  // namespace tdma
