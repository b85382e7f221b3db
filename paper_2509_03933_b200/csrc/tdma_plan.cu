// C-ABI implementation (include/tdma.h): plan management, the batch-pipeline scheduler
// (Alg. 2, re-expressed with CUDA events instead of cudaStreamSynchronize),
// CUDA-graph capture of the schedule, stage-isolated entry point, host-buffer solve.
#include "../../include/tdma.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "tdma_stage_kernels.cuh"
#include "tdma_fused.cuh"
#define TDMA_FUSED_TMA_DISPATCH
#include "tdma_fused_tma.cuh"
#include "tdma_shared.h"
#include "tdma_staged.h"

#define TDMA_VERSION_NUM 10200

namespace {

thread_local char g_err[512] = "";
thread_local int g_err_code = TDMA_OK;

int set_err(int code, const char *fmt, ...)
{
    g_err_code = code;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

#define CUDA_TRY(expr)                                                                       \
    do {                                                                                     \
        cudaError_t e_ = (expr);                                                             \
        if (e_ != cudaSuccess)                                                               \
            return set_err(TDMA_ERR_CUDA, "%s failed: %s (%s:%d)", #expr,                    \
                           cudaGetErrorString(e_), __FILE__, __LINE__);                      \
    } while (0)

constexpr int kMaxLanes = 7;
constexpr int kMaxDepth = kMaxLanes + 2;
constexpr int kPrefetchRows = 4;  // U of the stage kernels

struct SlabPtrs {
    const double *a, *b, *c, *d;
    double *x;
};

struct GraphEntry {
    SlabPtrs ptr;
    int nz;
    cudaGraphExec_t exec;
    unsigned long long stamp;
};

}  // namespace

struct tdma_plan {
    int nx = 0, ny = 0, nz = 0, P = 0, m = 0, bz = 0, nb = 0;
    int variant = TDMA_VARIANT_PIPELINED, nstreams = 2, nlanes = 1, depth = 3;
    int batch_arg = 0;                     // `batch` as passed to tdma_plan_create
    int use_graph = 1, separate_gather = 0;
    int pdd = 0;                           // stage B = PDD (far spike ends dropped, 2 x 2 interface systems)
    int timeline = 0;                      // timing events around every stage launch
    std::vector<cudaEvent_t> tl_ev;        // 2 per launch, reused across solves
    std::vector<int> tl_tag;               // stage * 2^20 + batch, per launch of the last solve
    int device = 0;
    // Inside the plan ny is the line length (rows along the solve axis) and nz the number of slices
    // (the other axis); for a z sweep they are the caller's nz and ny.
    int axis = TDMA_AXIS_Y, periodic = 0;
    long long rs = 0, os = 0;  // caller arrays: element stride between rows / between slices
    size_t slice = 0;   // nx * ny: one slice of the plan's scratch
    size_t Lb_max = 0;  // nx * bz
    size_t workspace = 0;
    // PIPELINED buffers (ring of `depth` slots)
    double *scratch = nullptr;  // depth x {SA, SC, SD} x [bz][ny][nx]
    double *red = nullptr;      // depth x {RA, RC, RD, CP, Y} x [2P][Lb_max]
    double *send = nullptr;     // depth x [P][6][Lb_max]            (separate_gather)
    cudaStream_t sMain = nullptr, sB = nullptr, lane[kMaxLanes] = {};
    cudaEvent_t evFork = nullptr, evBJoin = nullptr, evLaneJoin[kMaxLanes] = {};
    cudaEvent_t evA[kMaxDepth] = {}, evB[kMaxDepth] = {}, evC[kMaxDepth] = {};
    std::vector<GraphEntry> graphs;
    unsigned long long stamp = 0;
    int graph_builds = 0;
    // FUSED
    tdma::FusedConfig fused;
    int fused_impl = 0;  // 1 = register-staged general tree, 2 = TMA / pairwise tree
    tdma::TmaFusedConfig tfused;
    tdma::TmaFusedConfig tfill;   // clusters of <= 2 CTAs for the SMs the main launch cannot use
    bool have_fill = false;
    int fill_opt = 0, fill_last = 0, sm_count = 0;
    size_t sm_smem = 0;
    // STAGED: stage A / C as TMA-staged kernels, reduced system of Pred partitions in HBM
    tdma::StagedConfig staged;
    int Pred = 0;       // partitions in the reduced buffers (P; STAGED: staged.Pe)
    // shared-coefficient mode (tdma_solve_shared), configured at the first call per ncomp
    tdma::SharedConfig sh[3], sh_fill[3];   // real, complex, real with a uniform matrix (no shift arrays)
    int sh_state[3] = {0, 0, 0};  // 0 = not configured, 1 = ready, -1 = does not tile
    bool sh_have_fill[3] = {false, false, false};
    double *sh_zero = nullptr;    // zero shifts, for uniform-matrix calls on shapes the uniform tiling does not cover
    int sh_opt[5] = {0, 0, 0, 0, 0}; // options.shared_lines / _cluster / _leaf_rows / _slots / _ctas
    int sh_last = -1, sh_fill_last = 0;
    double *sh_lines = nullptr;        // scratch of the general-shape shared kernel (c', h' of a chunk of slices)
    size_t sh_lines_doubles = 0;
    int sh_lines_last = 0;             // 1: the last tdma_solve_shared ran the general-shape kernel
    // host staging (tdma_solve_host), allocated on first use
    int hz = 0;  // slices per host chunk
    tdma_options opt_saved = {};       // the options the plan was created with (struct_size = 0: none)
    tdma_plan *zchild[2] = {};         // tdma_solve_host of a z sweep: plans for a chunk of hz y-slices / the last, shorter chunk
    int host_chunk = 0;  // options.host_chunk (0 = auto)
    double *stage_dev[2][5] = {};
    cudaStream_t sH2D = nullptr, sD2H = nullptr;
    cudaEvent_t evH2D[2] = {}, evDone[2] = {}, evD2H[2] = {};
};

namespace {

double *slot_scratch(const tdma_plan *pl, int slot, int which)
{
    const size_t per = (size_t)pl->bz * pl->slice;
    return pl->scratch + ((size_t)slot * 3 + which) * per;
}
double *slot_red(const tdma_plan *pl, int slot, int which)
{
    const size_t per = (size_t)2 * pl->Pred * pl->Lb_max;
    return pl->red + ((size_t)slot * 5 + which) * per;
}

tdma::StageParams batch_params(const tdma_plan *pl, const SlabPtrs &ptr, int nz_count, int n)
{
    const int k0 = n * pl->bz;
    const int bzn = std::min(pl->bz, nz_count - k0);
    const int slot = n % pl->depth;
    const size_t off = (size_t)k0 * (size_t)pl->os;
    tdma::StageParams prm;
    prm.a = ptr.a + off; prm.b = ptr.b + off; prm.c = ptr.c + off; prm.d = ptr.d + off;
    prm.x = ptr.x + off;
    prm.sa = slot_scratch(pl, slot, 0); prm.sc = slot_scratch(pl, slot, 1);
    prm.sd = slot_scratch(pl, slot, 2);
    prm.ra = slot_red(pl, slot, 0); prm.rc = slot_red(pl, slot, 1); prm.rd = slot_red(pl, slot, 2);
    prm.cp = slot_red(pl, slot, 3); prm.y = slot_red(pl, slot, 4);
    prm.send = pl->send ? pl->send + (size_t)slot * 6 * pl->P * pl->Lb_max : nullptr;
    prm.Lb = (long long)pl->nx * bzn;
    prm.nx = pl->nx; prm.ny = pl->ny; prm.m = pl->m; prm.P = pl->P;
    prm.rs = pl->rs; prm.os = pl->os;
    if (pl->axis == TDMA_AXIS_X) { prm.rs = 1; prm.ls = pl->ny; }   // lines along the contiguous axis
    prm.pg0 = 0; prm.Ptot = pl->P; prm.Ls = 0;
    prm.cyclic = pl->periodic ? 1 : 0;
    return prm;
}

int launch_stage(tdma_plan *pl, int stage, const tdma::StageParams &prm_in, cudaStream_t st)
{
    tdma::StageParams prm = prm_in;
    const unsigned Lb = (unsigned)prm.Lb;
    if (pl->variant == TDMA_VARIANT_STAGED) {
        if (stage == TDMA_STAGE_A || stage == TDMA_STAGE_C) {
            const int nzs = (int)(prm.Lb / pl->nx);
            cudaError_t e = tdma::launch_staged(pl->staged, stage == TDMA_STAGE_A ? 1 : 2, prm.a, prm.b, prm.c, prm.d, prm.x,
                                                prm.ra, prm.rc, prm.rd, prm.y, pl->nx, pl->ny, nzs, pl->rs, pl->os,
                                                pl->axis == TDMA_AXIS_Z, st, pl->periodic != 0);
            if (e != cudaSuccess) return set_err(TDMA_ERR_CUDA, "staged launch failed: %s", cudaGetErrorString(e));
            return TDMA_OK;
        }
        if (stage == TDMA_STAGE_GATHER) return set_err(TDMA_ERR_INVALID_ARG, "STAGED plans have no separate gather stage");
        prm.P = pl->Pred;               // stage B: 2 Pred rows
    }
    switch (stage) {
    case TDMA_STAGE_A: {
        dim3 grid((Lb + 127) / 128, pl->P);
        if (pl->separate_gather)
            tdma::stage_a_kernel<kPrefetchRows, tdma::kOutSendA><<<grid, 128, 0, st>>>(prm);
        else
            tdma::stage_a_kernel<kPrefetchRows, tdma::kOutReduced><<<grid, 128, 0, st>>>(prm);
        break;
    }
    case TDMA_STAGE_GATHER: {
        dim3 grid((Lb + 255) / 256, pl->P);
        tdma::gather_kernel<<<grid, 256, 0, st>>>(prm);
        break;
    }
    case TDMA_STAGE_B:
        if (pl->pdd) {
            dim3 grid((Lb + 127) / 128, prm.P);
            tdma::stage_b_pdd_kernel<<<grid, 128, 0, st>>>(prm);
        } else if (pl->periodic) {
            tdma::stage_b_cyclic_kernel<<<(Lb + 63) / 64, 64, 0, st>>>(prm);
        } else {
            tdma::stage_b_kernel<kPrefetchRows><<<(Lb + 63) / 64, 64, 0, st>>>(prm);
        }
        break;
    case TDMA_STAGE_C: {
        dim3 grid((Lb + 127) / 128, pl->P);
        tdma::stage_c_kernel<kPrefetchRows><<<grid, 128, 0, st>>>(prm);
        break;
    }
    default:
        return set_err(TDMA_ERR_INVALID_ARG, "unknown stage %d", stage);
    }
    CUDA_TRY(cudaGetLastError());
    return TDMA_OK;
}

// Alg. 2 with events.  Iteration n enqueues A(n) on an A+C lane, B(n-1) on the B stream and
// C(n-2) on the lane that ran A(n-2); indices outside [0, nb) are skipped.
// Ring slot of batch n is n % depth with depth = nlanes + 2 >= 3 ("three batched systems
// concurrently"): A(n) may only overwrite a slot after C(n - depth) has read it.
int enqueue_pipelined(tdma_plan *pl, const SlabPtrs &ptr, int nz_count, cudaStream_t origin)
{
    if (pl->ny == 1) {
        const size_t n = (size_t)pl->nx * nz_count;
        tdma::diagonal_kernel<<<(unsigned)((n + 255) / 256), 256, 0, origin>>>(ptr.b, ptr.d, ptr.x, n);
        CUDA_TRY(cudaGetLastError());
        return TDMA_OK;
    }
    const int nb = (nz_count + pl->bz - 1) / pl->bz;
    int rc;
    if (pl->timeline) pl->tl_tag.clear();
    // stage launch, bracketed by timing events when the plan records a timeline
    auto run_stage = [&](int stage, const tdma::StageParams &prm, cudaStream_t st, int batch) -> int {
        if (!pl->timeline) return launch_stage(pl, stage, prm, st);
        const size_t i = pl->tl_tag.size();
        while (pl->tl_ev.size() < 2 * (i + 1)) {
            cudaEvent_t ev = nullptr;
            if (cudaEventCreate(&ev) != cudaSuccess) return set_err(TDMA_ERR_CUDA, "cudaEventCreate failed");
            pl->tl_ev.push_back(ev);
        }
        cudaEventRecord(pl->tl_ev[2 * i], st);
        const int r = launch_stage(pl, stage, prm, st);
        cudaEventRecord(pl->tl_ev[2 * i + 1], st);
        pl->tl_tag.push_back(stage * (1 << 20) + batch);
        return r;
    };
    if (pl->nstreams == 1) {  // Alg. 1 order: A, [A2B], B, C per batch
        for (int n = 0; n < nb; ++n) {
            const tdma::StageParams prm = batch_params(pl, ptr, nz_count, n);
            if ((rc = run_stage(TDMA_STAGE_A, prm, origin, n))) return rc;
            if (pl->separate_gather && (rc = run_stage(TDMA_STAGE_GATHER, prm, origin, n))) return rc;
            if ((rc = run_stage(TDMA_STAGE_B, prm, origin, n))) return rc;
            if ((rc = run_stage(TDMA_STAGE_C, prm, origin, n))) return rc;
        }
        return TDMA_OK;
    }
    CUDA_TRY(cudaEventRecord(pl->evFork, origin));
    for (int i = 0; i < pl->nlanes; ++i) CUDA_TRY(cudaStreamWaitEvent(pl->lane[i], pl->evFork, 0));
    CUDA_TRY(cudaStreamWaitEvent(pl->sB, pl->evFork, 0));
    for (int n = 0; n < nb + 2; ++n) {
        if (n < nb) {  // Stage A (n)
            const int slot = n % pl->depth;
            cudaStream_t st = pl->lane[n % pl->nlanes];
            if (n >= pl->depth) CUDA_TRY(cudaStreamWaitEvent(st, pl->evC[slot], 0));
            const tdma::StageParams prm = batch_params(pl, ptr, nz_count, n);
            if ((rc = run_stage(TDMA_STAGE_A, prm, st, n))) return rc;
            CUDA_TRY(cudaEventRecord(pl->evA[slot], st));
        }
        if (n - 1 >= 0 && n - 1 < nb) {  // Stage A2B + B (n-1)
            const int q = n - 1, slot = q % pl->depth;
            const tdma::StageParams prm = batch_params(pl, ptr, nz_count, q);
            CUDA_TRY(cudaStreamWaitEvent(pl->sB, pl->evA[slot], 0));
            if (pl->separate_gather && (rc = run_stage(TDMA_STAGE_GATHER, prm, pl->sB, q))) return rc;
            if ((rc = run_stage(TDMA_STAGE_B, prm, pl->sB, q))) return rc;
            CUDA_TRY(cudaEventRecord(pl->evB[slot], pl->sB));
        }
        if (n - 2 >= 0 && n - 2 < nb) {  // Stage B2C + C (n-2): C reads Y in place, no scatter
            const int q = n - 2, slot = q % pl->depth;
            cudaStream_t st = pl->lane[q % pl->nlanes];
            const tdma::StageParams prm = batch_params(pl, ptr, nz_count, q);
            CUDA_TRY(cudaStreamWaitEvent(st, pl->evB[slot], 0));
            if ((rc = run_stage(TDMA_STAGE_C, prm, st, q))) return rc;
            CUDA_TRY(cudaEventRecord(pl->evC[slot], st));
        }
    }
    for (int i = 0; i < pl->nlanes; ++i) {
        CUDA_TRY(cudaEventRecord(pl->evLaneJoin[i], pl->lane[i]));
        CUDA_TRY(cudaStreamWaitEvent(origin, pl->evLaneJoin[i], 0));
    }
    CUDA_TRY(cudaEventRecord(pl->evBJoin, pl->sB));
    CUDA_TRY(cudaStreamWaitEvent(origin, pl->evBJoin, 0));
    return TDMA_OK;
}

int enqueue_fused(tdma_plan *pl, const SlabPtrs &ptr, int nz_count, cudaStream_t origin)
{
    if (pl->ny == 1) return enqueue_pipelined(pl, ptr, nz_count, origin);
    // batches are contiguous z ranges; consecutive launches on one stream overlap their tails
    // only through the hardware's block scheduler, so by default one launch covers all slices
    const int nb = (nz_count + pl->bz - 1) / pl->bz;
    for (int n = 0; n < nb; ++n) {
        const int k0 = n * pl->bz;
        const int bzn = std::min(pl->bz, nz_count - k0);
        const size_t off = (size_t)k0 * (size_t)pl->os;
        const bool az = pl->axis == TDMA_AXIS_Z, per = pl->periodic != 0;
        const bool plain_y = pl->axis == TDMA_AXIS_Y && !per;
        cudaError_t e;
        const bool aligned = ((((uintptr_t)ptr.a | (uintptr_t)ptr.b | (uintptr_t)ptr.c | (uintptr_t)ptr.d |
                                (uintptr_t)ptr.x) & 15) == 0);   // tensor maps
        if (pl->fused_impl == 2 && aligned) {
            // Fill launch: a cluster of >= 4 CTAs cannot be placed on every SM.  With one main CTA
            // per SM the SMs left over take a second persistent launch with clusters of 2 that
            // solves the last nzf slices concurrently (forked from / joined to `origin`).
            int nzf = 0;
            if (pl->have_fill) {
                e = tdma::launch_tma_fused(pl->tfused, ptr.a, ptr.b, ptr.c, ptr.d, ptr.x, pl->nx, pl->ny, 0, pl->rs, pl->os, az, per, origin);
                if (e == cudaSuccess)
                    e = tdma::launch_tma_fused(pl->tfill, ptr.a, ptr.b, ptr.c, ptr.d, ptr.x, pl->nx, pl->ny, 0, pl->rs, pl->os, az, per, origin);
                if (e != cudaSuccess)
                    return set_err(TDMA_ERR_CUDA, "fused launch preparation failed: %s", cudaGetErrorString(e));
                const long per_sm = (long)(pl->sm_smem / (pl->tfused.smem + 1024));
                const int main_ctas = pl->tfused.max_clusters * pl->tfused.cluster;
                const int idle = per_sm == 1 ? pl->sm_count - main_ctas : 0;
                int fc = idle / pl->tfill.cluster;
                if (fc > pl->tfill.max_clusters) fc = pl->tfill.max_clusters;
                if (fc > 0) {
                    // measured: with 64-byte row segments in the fill tiling (cfg 3: 8 lines per tile,
                    // neighbouring x tiles taken in pairs) the step time is flat for shares of 8-12 of
                    // 128 slices (6.97-7.04 ms); the smallest of them, weight 0.55, leaves the most to
                    // the main launch.  With 128-byte segments a fill SM does as much as a main SM
                    // (cfg 4 z sweeps: best share 0.11 = 16 / 148 SMs)
                    const double w = (pl->tfill.lines >= 16 ? 1.0 : 0.55) * fc * pl->tfill.cluster;
                    double share = pl->fill_opt > 0 ? pl->fill_opt * 1e-3 : w / (w + main_ctas);
                    nzf = (int)(bzn * share + 0.5);
                    if (nzf >= bzn) nzf = bzn - 1;
                    if (nzf > 0) pl->tfill.max_clusters = fc;     // never more than the idle SMs
                }
            }
            pl->fill_last = nzf;
            if (nzf > 0) {
                CUDA_TRY(cudaEventRecord(pl->evFork, origin));
                CUDA_TRY(cudaStreamWaitEvent(pl->sB, pl->evFork, 0));
            }
            e = tdma::launch_tma_fused(pl->tfused, ptr.a + off, ptr.b + off, ptr.c + off, ptr.d + off,
                                       ptr.x + off, pl->nx, pl->ny, bzn - nzf, pl->rs, pl->os, az, per, origin);
            if (e == cudaSuccess && nzf > 0) {
                const size_t offf = off + (size_t)(bzn - nzf) * (size_t)pl->os;
                e = tdma::launch_tma_fused(pl->tfill, ptr.a + offf, ptr.b + offf, ptr.c + offf, ptr.d + offf,
                                           ptr.x + offf, pl->nx, pl->ny, nzf, pl->rs, pl->os, az, per, pl->sB);
                // join even when the fill launch failed: `origin` must not be left forked
                cudaError_t ej = cudaEventRecord(pl->evBJoin, pl->sB);
                if (ej == cudaSuccess) ej = cudaStreamWaitEvent(origin, pl->evBJoin, 0);
                if (e == cudaSuccess) e = ej;
            }
        } else if (pl->fused.threads > 0 && plain_y)
            e = tdma::launch_fused(pl->fused, ptr.a + off, ptr.b + off, ptr.c + off,
                                   ptr.d + off, ptr.x + off, pl->nx, pl->ny, bzn, origin);
        else
            return set_err(TDMA_ERR_UNSUPPORTED, "fused TMA kernel needs 16-byte aligned arrays%s",
                           plain_y ? "" : " (x / z sweeps and cyclic lines of such arrays: TDMA_VARIANT_PIPELINED)");
        if (e != cudaSuccess)
            return set_err(TDMA_ERR_CUDA, "fused launch failed: %s", cudaGetErrorString(e));
    }
    return TDMA_OK;
}

int enqueue_schedule(tdma_plan *pl, const SlabPtrs &ptr, int nz_count, cudaStream_t origin)
{
    return pl->variant == TDMA_VARIANT_FUSED ? enqueue_fused(pl, ptr, nz_count, origin)
                                             : enqueue_pipelined(pl, ptr, nz_count, origin);
}

int launches_per_solve(const tdma_plan *pl)
{
    if (pl->ny == 1) return 1;
    if (pl->variant == TDMA_VARIANT_FUSED) return pl->nb * (pl->fill_last > 0 ? 2 : 1);   // after a solve: main + fill launch
    return pl->nb * (3 + (pl->separate_gather ? 1 : 0));
}

// Look up / build the CUDA graph of the whole schedule for this pointer set.
int graph_for(tdma_plan *pl, const SlabPtrs &ptr, int nz_count, cudaGraphExec_t *out)
{
    for (auto &g : pl->graphs)
        if (g.nz == nz_count && g.ptr.a == ptr.a && g.ptr.b == ptr.b && g.ptr.c == ptr.c &&
            g.ptr.d == ptr.d && g.ptr.x == ptr.x) {
            g.stamp = ++pl->stamp;
            *out = g.exec;
            return TDMA_OK;
        }
    cudaGraph_t graph = nullptr;
    CUDA_TRY(cudaStreamBeginCapture(pl->sMain, cudaStreamCaptureModeThreadLocal));
    int rc = enqueue_schedule(pl, ptr, nz_count, pl->sMain);
    cudaError_t e = cudaStreamEndCapture(pl->sMain, &graph);
    if (rc != TDMA_OK) {
        if (graph) cudaGraphDestroy(graph);
        return rc;
    }
    if (e != cudaSuccess)
        return set_err(TDMA_ERR_CUDA, "cudaStreamEndCapture failed: %s", cudaGetErrorString(e));
    cudaGraphExec_t exec = nullptr;
    e = cudaGraphInstantiate(&exec, graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess)
        return set_err(TDMA_ERR_CUDA, "cudaGraphInstantiate failed: %s", cudaGetErrorString(e));
    if (pl->graphs.size() >= 8) {  // evict least recently used
        auto it = std::min_element(pl->graphs.begin(), pl->graphs.end(),
                                   [](const GraphEntry &x, const GraphEntry &y) { return x.stamp < y.stamp; });
        cudaGraphExecDestroy(it->exec);
        pl->graphs.erase(it);
    }
    pl->graphs.push_back(GraphEntry{ptr, nz_count, exec, ++pl->stamp});
    pl->graph_builds++;
    *out = exec;
    return TDMA_OK;
}

int run_solve(tdma_plan *pl, const SlabPtrs &ptr, int nz_count, cudaStream_t stream)
{
    if (pl->use_graph) {
        cudaGraphExec_t exec = nullptr;
        int rc = graph_for(pl, ptr, nz_count, &exec);
        if (rc != TDMA_OK) return rc;
        CUDA_TRY(cudaGraphLaunch(exec, stream));
        return TDMA_OK;
    }
    return enqueue_schedule(pl, ptr, nz_count, stream);
}

void free_plan(tdma_plan *pl)
{
    if (!pl) return;
    for (auto &g : pl->graphs) cudaGraphExecDestroy(g.exec);
    for (auto ev : pl->tl_ev) cudaEventDestroy(ev);
    cudaFree(pl->scratch); cudaFree(pl->red); cudaFree(pl->send); cudaFree(pl->sh_zero); cudaFree(pl->sh_lines);
    if (pl->staged.impl) tdma::free_staged(&pl->staged);
    for (int s = 0; s < 2; ++s)
        for (int i = 0; i < 5; ++i) cudaFree(pl->stage_dev[s][i]);
    free_plan(pl->zchild[0]); free_plan(pl->zchild[1]);
    auto ds = [](cudaStream_t s) { if (s) cudaStreamDestroy(s); };
    auto de = [](cudaEvent_t e) { if (e) cudaEventDestroy(e); };
    ds(pl->sMain); ds(pl->sB); ds(pl->sH2D); ds(pl->sD2H);
    for (int i = 0; i < kMaxLanes; ++i) { ds(pl->lane[i]); de(pl->evLaneJoin[i]); }
    for (int i = 0; i < kMaxDepth; ++i) { de(pl->evA[i]); de(pl->evB[i]); de(pl->evC[i]); }
    for (int i = 0; i < 2; ++i) { de(pl->evH2D[i]); de(pl->evDone[i]); de(pl->evD2H[i]); }
    de(pl->evFork); de(pl->evBJoin);
    delete pl;
}

int init_plan(tdma_plan *pl, const tdma_options *opt)
{
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev < 1)
        return set_err(TDMA_ERR_CUDA, "no CUDA device (%s); this library has no CPU fallback",
                       e != cudaSuccess ? cudaGetErrorString(e) : "device count is 0");
    CUDA_TRY(cudaGetDevice(&pl->device));
    cudaDeviceProp prop;
    CUDA_TRY(cudaGetDeviceProperties(&prop, pl->device));
    if (prop.major < 10)
        return set_err(TDMA_ERR_UNSUPPORTED, "device sm_%d%d: this build targets sm_100a only",
                       prop.major, prop.minor);

    int variant = opt ? opt->variant : 0;
    if (variant == TDMA_VARIANT_AUTO) {
        // the fastest path that can run this plan: the fused TMA kernel in ONE persistent launch
        // (batch is then only a hint for the pipelined variant), else the stage pipeline
        tdma::TmaFusedConfig probe;
        const char *why = nullptr;
        const bool tma_ok = pl->ny > 1 && tdma::get_encode_tiled() != nullptr &&
                            tdma::configure_tma_fused(&probe, pl->nx, pl->ny, pl->P, opt ? opt->fused_lines : 0,
                                                      opt ? opt->fused_cluster : 0, opt ? opt->fused_leaf_rows : 0,
                                                      prop, &why, pl->axis == TDMA_AXIS_X, pl->axis == TDMA_AXIS_Z,
                                                      opt ? opt->fused_slots : 0);
        variant = tma_ok ? TDMA_VARIANT_FUSED : TDMA_VARIANT_PIPELINED;
        if (variant == TDMA_VARIANT_FUSED) pl->batch_arg = 0;   // batch is a hint for the stage pipelines only
    }
    if (variant == TDMA_VARIANT_FUSED && pl->batch_arg == 0) {
        // FUSED default: launches of about 2^27 cells (128 slices of 1024 x 1024).  The clusters of a
        // persistent launch drift apart over a long run and DRAM row locality between neighbouring
        // x tiles goes with it; a fresh launch every ~0.9 ms re-aligns them (measured on cfg 3:
        // 7.25 ms as one launch, 7.02 ms in chunks of 128-256 slices; cfg 5: 7.38 -> 7.22 ms)
        const long long chunk = std::max<long long>(1, ((long long)1 << 27) / (long long)pl->slice);
        pl->bz = (int)std::min<long long>(pl->nz, chunk);
        pl->nb = (pl->nz + pl->bz - 1) / pl->bz;
        pl->Lb_max = (size_t)pl->nx * pl->bz;
    }
    if (variant != TDMA_VARIANT_PIPELINED && variant != TDMA_VARIANT_FUSED && variant != TDMA_VARIANT_STAGED)
        return set_err(TDMA_ERR_INVALID_ARG, "unknown variant %d", variant);
    if (variant == TDMA_VARIANT_STAGED && (pl->axis == TDMA_AXIS_X || pl->ny < 2))
        return set_err(TDMA_ERR_UNSUPPORTED, "the STAGED variant does y / z sweeps of lines with >= 2 rows");
    if (pl->periodic && pl->ny < 2)
        return set_err(TDMA_ERR_UNSUPPORTED, "cyclic lines need >= 2 rows");
    if (pl->periodic && opt && opt->pdd > 0)
        return set_err(TDMA_ERR_UNSUPPORTED, "pdd is defined for plain lines only");
    pl->variant = variant;
    pl->Pred = pl->P;
    pl->use_graph = (opt && opt->use_graph < 0) ? 0 : 1;
    pl->timeline = (opt && opt->timeline > 0) ? 1 : 0;
    if (pl->timeline) pl->use_graph = 0;
    pl->separate_gather = (opt && opt->separate_gather > 0) ? 1 : 0;
    pl->pdd = (opt && opt->pdd > 0) ? 1 : 0;
    if (pl->pdd && variant == TDMA_VARIANT_FUSED)
        return set_err(TDMA_ERR_UNSUPPORTED, "pdd replaces stage B of the PIPELINED / STAGED variants; FUSED has no separate stage B");
    pl->nstreams = (opt && opt->nstreams > 0) ? opt->nstreams : 2;
    if (pl->nstreams > kMaxLanes + 1)
        return set_err(TDMA_ERR_INVALID_ARG, "nstreams %d > %d", pl->nstreams, kMaxLanes + 1);
    pl->nlanes = std::max(1, pl->nstreams - 1);
    pl->depth = pl->nstreams == 1 ? 1 : pl->nlanes + 2;

    int lo = 0, hi = 0;  // stage B's stream gets the highest priority so its small kernels are
    CUDA_TRY(cudaDeviceGetStreamPriorityRange(&lo, &hi));  // scheduled as soon as SM slots free up
    CUDA_TRY(cudaStreamCreateWithPriority(&pl->sMain, cudaStreamNonBlocking, lo));
    CUDA_TRY(cudaStreamCreateWithPriority(&pl->sB, cudaStreamNonBlocking, hi));
    for (int i = 0; i < pl->nlanes; ++i)
        CUDA_TRY(cudaStreamCreateWithPriority(&pl->lane[i], cudaStreamNonBlocking, lo));
    auto mk = [](cudaEvent_t *ev) { return cudaEventCreateWithFlags(ev, cudaEventDisableTiming); };
    CUDA_TRY(mk(&pl->evFork)); CUDA_TRY(mk(&pl->evBJoin));
    for (int i = 0; i < pl->nlanes; ++i) CUDA_TRY(mk(&pl->evLaneJoin[i]));
    for (int i = 0; i < pl->depth; ++i) { CUDA_TRY(mk(&pl->evA[i])); CUDA_TRY(mk(&pl->evB[i])); CUDA_TRY(mk(&pl->evC[i])); }

    if (variant == TDMA_VARIANT_STAGED) {
        const char *why = nullptr;
        if (!tdma::configure_staged(&pl->staged, pl->nx, pl->ny, pl->P, pl->axis == TDMA_AXIS_Z, prop, &why))
            return set_err(TDMA_ERR_UNSUPPORTED, "STAGED variant unavailable: %s", why ? why : "?");
        pl->Pred = pl->staged.Pe;
        if (opt && opt->separate_gather > 0) return set_err(TDMA_ERR_UNSUPPORTED, "STAGED plans fuse the gather into stage A");
        const size_t rbytes = (size_t)pl->depth * 5 * 2 * pl->Pred * pl->Lb_max * sizeof(double);
        if (cudaMalloc(&pl->red, rbytes) != cudaSuccess) {
            cudaGetLastError();
            return set_err(TDMA_ERR_ALLOC, "cannot allocate %zu bytes of reduced-system ring", rbytes);
        }
        pl->workspace = rbytes;
    }
    if (variant == TDMA_VARIANT_PIPELINED && pl->ny > 1) {
        const size_t sbytes = (size_t)pl->depth * 3 * pl->bz * pl->slice * sizeof(double);
        const size_t rbytes = (size_t)pl->depth * 5 * 2 * pl->P * pl->Lb_max * sizeof(double);
        if (cudaMalloc(&pl->scratch, sbytes) != cudaSuccess || cudaMalloc(&pl->red, rbytes) != cudaSuccess) {
            cudaGetLastError();
            return set_err(TDMA_ERR_ALLOC, "cannot allocate %zu bytes of scratch ring", sbytes + rbytes);
        }
        pl->workspace = sbytes + rbytes;
        if (pl->separate_gather) {
            const size_t gbytes = (size_t)pl->depth * 6 * pl->P * pl->Lb_max * sizeof(double);
            if (cudaMalloc(&pl->send, gbytes) != cudaSuccess) {
                cudaGetLastError();
                return set_err(TDMA_ERR_ALLOC, "cannot allocate %zu bytes of send_A buffer", gbytes);
            }
            pl->workspace += gbytes;
        }
    }
    if (variant == TDMA_VARIANT_FUSED && pl->ny > 1) {
        const char *why = nullptr;
        if ((size_t)pl->nx * (size_t)pl->m >= ((size_t)1 << 32))
            return set_err(TDMA_ERR_UNSUPPORTED, "fused variant: nx * ny/P exceeds 2^32 elements");
        int want_impl = opt ? opt->fused_impl : 0;
        if (want_impl < 0 || want_impl > 2)
            return set_err(TDMA_ERR_INVALID_ARG, "unknown fused_impl %d", want_impl);
        if (pl->axis != TDMA_AXIS_Y || pl->periodic) {
            if (want_impl == 1)
                return set_err(TDMA_ERR_UNSUPPORTED, "the register-staged fused kernel does y sweeps of plain lines only");
            want_impl = 2;
        }
        bool have_tma = false;
        if (want_impl != 1) {
            have_tma = tdma::get_encode_tiled() != nullptr &&
                       tdma::configure_tma_fused(&pl->tfused, pl->nx, pl->ny, pl->P, opt ? opt->fused_lines : 0,
                                                 opt ? opt->fused_cluster : 0, opt ? opt->fused_leaf_rows : 0,
                                                 prop, &why, pl->axis == TDMA_AXIS_X, pl->axis == TDMA_AXIS_Z,
                                                 opt ? opt->fused_slots : 0);
            if (!have_tma && want_impl == 2)
                return set_err(TDMA_ERR_UNSUPPORTED, "fused TMA kernel unavailable: %s",
                               why ? why : "cuTensorMapEncodeTiled not found");
        }
        // the register-staged kernel is the fallback for unaligned pointers (explicit options
        // are only forwarded to it when it was asked for)
        const bool fwd = want_impl == 1 || !have_tma;
        const bool have_reg = pl->axis == TDMA_AXIS_Y && !pl->periodic &&
                              tdma::configure_fused(&pl->fused, pl->nx, pl->ny, pl->P,
                                                    fwd && opt ? opt->fused_lines : 0,
                                                    fwd && opt ? opt->fused_cluster : 0,
                                                    fwd && opt ? opt->fused_leaf_rows : 0,
                                                    opt ? opt->fused_top : 0, prop, &why);
        if (!have_reg) pl->fused = tdma::FusedConfig();
        if (!have_tma && !have_reg)
            return set_err(TDMA_ERR_UNSUPPORTED, "fused variant unavailable: %s", why ? why : "?");
        pl->fused_impl = have_tma ? 2 : 1;
        pl->sm_count = prop.multiProcessorCount;
        pl->sm_smem = prop.sharedMemPerMultiprocessor;
        pl->fill_opt = opt ? opt->fused_fill : 0;
        // clusters of 5 / 6 (3 * 2^k, 5 * 2^k lines): no automatic fill launch -- the cluster-of-2 tiling of
        // such lengths is slow enough to finish last (ny = 640: 5.08 TB/s without it, 3.39 with it)
        const bool pow2_cluster = (pl->tfused.cluster & (pl->tfused.cluster - 1)) == 0;
        if (have_tma && pl->tfused.cluster >= 4 && pl->fill_opt >= 0 && (pow2_cluster || pl->fill_opt > 0)) {
            const char *why2 = nullptr;
            pl->have_fill = tdma::configure_tma_fused(&pl->tfill, pl->nx, pl->ny, pl->P, 0,
                                                      pl->ny % 2 == 0 ? 2 : 1, 0, prop, &why2,
                                                      pl->axis == TDMA_AXIS_X, pl->axis == TDMA_AXIS_Z);
        }
    }
    return TDMA_OK;
}

int check_ptrs(const tdma_plan *plan, const void *a, const void *b, const void *c, const void *d,
               const void *x)
{
    if (!plan) return set_err(TDMA_ERR_INVALID_ARG, "plan is NULL");
    if (!a || !b || !c || !d || !x) return set_err(TDMA_ERR_INVALID_ARG, "NULL array pointer");
    int dev = -1;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev != plan->device)
        return set_err(TDMA_ERR_INVALID_ARG, "plan was created on device %d, the current device is %d",
                       plan->device, dev);
    return TDMA_OK;
}

}  // namespace

namespace {

// tdma_solve_shared on shapes / alignments the tiled TMA kernel does not take: one thread per line
// (tdma_shared_lines.cu), the z range in chunks whose c' (and h' for cyclic lines) fit a plan-owned
// scratch array of at most 256 MiB (one slice, if a slice alone needs more), allocated at the first such call.
int shared_lines_solve(tdma_plan *pl, const void *a_y, const void *b0_y, const void *c_y, const void *sx, const void *sz,
                       int ncomp, int pin00, const void *d, void *x, cudaStream_t st)
{
    if (pl->periodic && pl->ny < 2) return set_err(TDMA_ERR_INVALID_ARG, "tdma_solve_shared: cyclic lines need >= 2 rows");
    const size_t per_slice = (size_t)pl->ny * (size_t)pl->nx * (pl->periodic ? 2 : 1);   // doubles of scratch
    const size_t budget = (size_t)32 << 20;
    long long sl = (long long)std::max<size_t>(1, budget / per_slice);
    if (sl > pl->nz) sl = pl->nz;
    const size_t need = per_slice * (size_t)sl;
    if (need > pl->sh_lines_doubles) {
        cudaFree(pl->sh_lines);
        pl->sh_lines = nullptr; pl->sh_lines_doubles = 0;
        if (cudaMalloc(&pl->sh_lines, need * sizeof(double)) != cudaSuccess) {
            cudaGetLastError();
            return set_err(TDMA_ERR_ALLOC, "tdma_solve_shared: cannot allocate %zu bytes of line scratch", need * sizeof(double));
        }
        pl->sh_lines_doubles = need;
    }
    tdma::SharedLineArgs args;
    args.a_y = (const double *)a_y; args.b0_y = (const double *)b0_y; args.c_y = (const double *)c_y;
    args.sx = (const double *)sx; args.sz = (const double *)sz;
    args.n = pl->ny; args.lanes = pl->nx;
    args.ncomp = ncomp; args.pin00 = pin00 ? 1 : 0; args.periodic = pl->periodic ? 1 : 0;
    if (pl->axis == TDMA_AXIS_X) { args.rs = 1; args.ls = pl->ny; args.os = (long long)pl->nx * pl->ny; }
    else { args.rs = pl->rs; args.ls = 1; args.os = pl->os; }
    for (long long k0 = 0; k0 < pl->nz; k0 += sl) {
        const long long n = std::min<long long>(sl, pl->nz - k0);
        const size_t off = (size_t)k0 * (size_t)args.os * (size_t)ncomp;
        args.d = (const double *)d + off; args.x = (double *)x + off;
        args.k0 = (int)k0; args.slices = (int)n;
        args.cs = pl->sh_lines; args.hs = pl->sh_lines + (size_t)pl->ny * (size_t)pl->nx * (size_t)n;
        const cudaError_t e = tdma::launch_shared_lines(args, st);
        if (e != cudaSuccess) return set_err(TDMA_ERR_CUDA, "shared line-kernel launch failed: %s", cudaGetErrorString(e));
    }
    pl->sh_last = -1; pl->sh_fill_last = 0; pl->sh_lines_last = 1;
    return TDMA_OK;
}

}  // namespace

namespace tdma {
// for the library's other translation units: sets the calling thread's tdma_last_error() message
int report_error(int code, const char *msg) { return set_err(code, "%s", msg); }
}  // namespace tdma

extern "C" {

tdma_plan *tdma_plan_create_ex(int nx, int ny, int nz, int P, int batch, int dtype,
                               const tdma_options *options)
{
    g_err[0] = 0;
    if (options && options->struct_size != (int)sizeof(tdma_options)) { set_err(TDMA_ERR_INVALID_ARG, "tdma_options.struct_size = %d, expected %zu", options->struct_size, sizeof(tdma_options)); return nullptr; }
    const int axis = options ? options->axis : TDMA_AXIS_Y, periodic = options && options->periodic ? 1 : 0;
    if (axis != TDMA_AXIS_Y && axis != TDMA_AXIS_Z && axis != TDMA_AXIS_X) { set_err(TDMA_ERR_INVALID_ARG, "unknown axis %d", axis); return nullptr; }
    if (axis == TDMA_AXIS_Z) std::swap(ny, nz);   // from here on: ny = line length, nz = slices,
    if (axis == TDMA_AXIS_X) std::swap(nx, ny);   // nx = lanes (lines side by side in a tile)
    if (nx < 1 || ny < 1 || nz < 1) { set_err(TDMA_ERR_INVALID_ARG, "dimensions must be >= 1 (got %d x %d x %d)", nx, ny, nz); return nullptr; }
    if (P < 1) { set_err(TDMA_ERR_INVALID_ARG, "P must be >= 1 (got %d)", P); return nullptr; }
    if (ny % P != 0) { set_err(TDMA_ERR_INVALID_ARG, "ny = %d is not divisible by P = %d", ny, P); return nullptr; }
    if (P > 1 && ny / P < 2) { set_err(TDMA_ERR_INVALID_ARG, "partitions need >= 2 rows (ny/P = %d)", ny / P); return nullptr; }
    if (batch < 0 || batch > nz) { set_err(TDMA_ERR_INVALID_ARG, "batch = %d outside [0, nz = %d]", batch, nz); return nullptr; }
    if (dtype != TDMA_F64) { set_err(TDMA_ERR_UNSUPPORTED, "dtype %d: only TDMA_F64 is implemented", dtype); return nullptr; }
    if (options && options->fused_slots != 0 && (options->fused_slots < 4 || options->fused_slots > 8)) { set_err(TDMA_ERR_INVALID_ARG, "fused_slots = %d must be 0 or 4 .. 8", options->fused_slots); return nullptr; }
    if (options && options->host_chunk < 0) { set_err(TDMA_ERR_INVALID_ARG, "host_chunk = %d must be >= 0", options->host_chunk); return nullptr; }
    if ((long long)nx * (batch ? batch : nz) > 0x7fffffffLL) { set_err(TDMA_ERR_UNSUPPORTED, "nx * batch exceeds 2^31-1 lines per batch"); return nullptr; }
    tdma_plan *pl = new (std::nothrow) tdma_plan();
    if (!pl) { set_err(TDMA_ERR_ALLOC, "out of host memory"); return nullptr; }
    pl->nx = nx; pl->ny = ny; pl->nz = nz; pl->P = P; pl->m = ny / P;   // ny, nz already mapped
    pl->axis = axis; pl->periodic = periodic;
    if (options) pl->opt_saved = *options;
    pl->host_chunk = options ? options->host_chunk : 0;
    pl->fill_opt = options ? options->fused_fill : 0;
    if (options) { pl->sh_opt[0] = options->shared_lines; pl->sh_opt[1] = options->shared_cluster; pl->sh_opt[2] = options->shared_leaf_rows; pl->sh_opt[3] = options->shared_slots; pl->sh_opt[4] = options->shared_ctas; }
    pl->rs = axis == TDMA_AXIS_Z ? (long long)nx * nz : (long long)nx;   // z sweep: plan nz = caller ny
    pl->os = axis == TDMA_AXIS_Z ? (long long)nx : (long long)nx * ny;   // x sweep: slices are z-slices
    pl->batch_arg = batch;
    pl->bz = batch == 0 ? nz : batch;
    pl->nb = (nz + pl->bz - 1) / pl->bz;
    pl->slice = (size_t)nx * ny;
    pl->Lb_max = (size_t)nx * pl->bz;
    if (init_plan(pl, options) != TDMA_OK) { free_plan(pl); return nullptr; }
    return pl;
}

tdma_plan *tdma_plan_create(int nx, int ny, int nz, int P, int batch, int dtype)
{
    return tdma_plan_create_ex(nx, ny, nz, P, batch, dtype, nullptr);
}

int tdma_solve(tdma_plan *plan, const void *a, const void *b, const void *c, const void *d,
               void *x, void *stream)
{
    int rc = check_ptrs(plan, a, b, c, d, x);
    if (rc != TDMA_OK) return rc;
    const SlabPtrs ptr{(const double *)a, (const double *)b, (const double *)c, (const double *)d, (double *)x};
    return run_solve(plan, ptr, plan->nz, (cudaStream_t)stream);
}

int tdma_stage(tdma_plan *plan, int stage, int batch_index, const void *a, const void *b,
               const void *c, const void *d, void *x, void *stream)
{
    int rc = check_ptrs(plan, a, b, c, d, x);
    if (rc != TDMA_OK) return rc;
    if ((plan->variant != TDMA_VARIANT_PIPELINED && plan->variant != TDMA_VARIANT_STAGED) || plan->ny == 1)
        return set_err(TDMA_ERR_UNSUPPORTED, "tdma_stage needs a PIPELINED or STAGED plan with ny > 1");
    if (batch_index < 0 || batch_index >= plan->nb)
        return set_err(TDMA_ERR_INVALID_ARG, "batch_index %d outside [0, %d)", batch_index, plan->nb);
    if (stage == TDMA_STAGE_GATHER && !plan->separate_gather)
        return set_err(TDMA_ERR_INVALID_ARG, "plan has no separate gather stage");
    const SlabPtrs ptr{(const double *)a, (const double *)b, (const double *)c, (const double *)d, (double *)x};
    const tdma::StageParams prm = batch_params(plan, ptr, plan->nz, batch_index);
    return launch_stage(plan, stage, prm, (cudaStream_t)stream);
}

int tdma_solve_shared(tdma_plan *plan, const void *a_y, const void *b0_y, const void *c_y,
                      const void *sx, const void *sz, int ncomp, int pin00, const void *d, void *x,
                      void *stream)
{
    int rc = check_ptrs(plan, a_y, b0_y, c_y, d, x);
    if (rc != TDMA_OK) return rc;
    if (ncomp != 1 && ncomp != 2) return set_err(TDMA_ERR_INVALID_ARG, "ncomp = %d must be 1 (real) or 2 (complex)", ncomp);
    tdma_plan *pl = plan;
    bool uniform = !sx && !sz;                 // the same matrix for every line
    if (!uniform && (!sx || !sz)) return set_err(TDMA_ERR_INVALID_ARG, "NULL shift array (pass both as NULL for a uniform matrix)");
    if (uniform && pin00) return set_err(TDMA_ERR_INVALID_ARG, "tdma_solve_shared: pin00 changes one line's matrix; pass shift arrays");
    const bool xsw = pl->axis == TDMA_AXIS_X;
    cudaStream_t origin = (cudaStream_t)stream;
    if (pl->periodic && pin00)
        return set_err(TDMA_ERR_INVALID_ARG, "tdma_solve_shared: pin00 is for plain lines");
    if ((((uintptr_t)d | (uintptr_t)x) & 7) != 0)
        return set_err(TDMA_ERR_INVALID_ARG, "tdma_solve_shared: d and x must be 8-byte aligned");
    // What the tiled TMA kernel does not take goes to the one-thread-per-line kernel, unless the caller
    // asked for a particular tiling (then the refusal is the answer).
    const bool asked = pl->sh_opt[0] || pl->sh_opt[1] || pl->sh_opt[2] || pl->sh_opt[3] || pl->sh_opt[4];
    const void *sx_in = sx, *sz_in = sz;
    auto line_kernel = [&]() { return shared_lines_solve(pl, a_y, b0_y, c_y, sx_in, sz_in, ncomp, pin00, d, x, origin); };
    pl->sh_lines_last = 0;
    if (xsw && ncomp != 1) {
        if (!asked) return line_kernel();
        return set_err(TDMA_ERR_UNSUPPORTED, "tdma_solve_shared: the tiled x sweep takes real right-hand sides (ncomp = 1)");
    }
    if ((((uintptr_t)d | (uintptr_t)x) & 15) != 0) {
        if (!asked) return line_kernel();
        return set_err(TDMA_ERR_UNSUPPORTED, "tdma_solve_shared: the tiled kernel needs 16-byte aligned d and x (tensor maps)");
    }
    if (pl->ny == 1) {
        if (!asked) return line_kernel();
        return set_err(TDMA_ERR_UNSUPPORTED, "tdma_solve_shared: the tiled kernel needs ny >= 4");
    }
    if (uniform && ncomp == 1 && pl->sh_state[2] == 0) {
        // the uniform-matrix build covers 16-line tiles with 16- / 32-row leaves and up to 256 threads
        cudaDeviceProp prop;
        CUDA_TRY(cudaGetDeviceProperties(&prop, pl->device));
        const char *why = nullptr;
        const bool ok = tdma::configure_shared(&pl->sh[2], pl->nx, pl->ny, 1, pl->sh_opt[0], pl->sh_opt[1], pl->sh_opt[2],
                                               pl->sh_opt[3], 0, prop, &why, xsw, true);
        pl->sh_state[2] = ok ? 1 : -1;
        pl->sm_count = prop.multiProcessorCount;
        pl->sm_smem = prop.sharedMemPerMultiprocessor;
        if (ok && pl->sh[2].cluster >= 4 && pl->fill_opt >= 0) {
            const char *why2 = nullptr;
            pl->sh_have_fill[2] = tdma::configure_shared(&pl->sh_fill[2], pl->nx, pl->ny, 1, 0, pl->ny % 2 == 0 ? 2 : 1,
                                                         0, 0, 0, prop, &why2, xsw, true);
        }
    }
    if (uniform && (ncomp != 1 || pl->sh_state[2] < 0)) {
        // no uniform-matrix build for this shape / complex cells: the general form with zero shifts
        const size_t nzero = (size_t)std::max(std::max(pl->nx, pl->ny), pl->nz);
        if (!pl->sh_zero) {
            if (cudaMalloc(&pl->sh_zero, nzero * sizeof(double)) != cudaSuccess) {
                cudaGetLastError();
                return set_err(TDMA_ERR_ALLOC, "tdma_solve_shared: no memory for %zu zero shifts", nzero);
            }
            CUDA_TRY(cudaMemset(pl->sh_zero, 0, nzero * sizeof(double)));
        }
        sx = sz = pl->sh_zero;
        uniform = false;
    }
    const int q = uniform ? 2 : ncomp - 1;
    if (pl->sh_state[q] == 0) {
        cudaDeviceProp prop;
        CUDA_TRY(cudaGetDeviceProperties(&prop, pl->device));
        const char *why = nullptr;
        if (!tdma::configure_shared(&pl->sh[q], pl->nx, pl->ny, ncomp, pl->sh_opt[0], pl->sh_opt[1], pl->sh_opt[2],
                                    pl->sh_opt[3], pl->sh_opt[4], prop, &why, xsw)) {
            pl->sh_state[q] = -1;
            if (!asked) return line_kernel();
            return set_err(TDMA_ERR_UNSUPPORTED, "tdma_solve_shared unavailable for this shape: %s", why ? why : "?");
        }
        pl->sm_count = prop.multiProcessorCount;
        pl->sm_smem = prop.sharedMemPerMultiprocessor;
        if (pl->sh[q].cluster >= 4 && pl->fill_opt >= 0) {
            const char *why2 = nullptr;
            pl->sh_have_fill[q] = tdma::configure_shared(&pl->sh_fill[q], pl->nx, pl->ny, ncomp, 0,
                                                         pl->ny % 2 == 0 ? 2 : 1, 0, 0, 0, prop, &why2, xsw);
        }
        pl->sh_state[q] = 1;
    }
    if (pl->sh_state[q] < 0) {
        if (!asked) return line_kernel();
        return set_err(TDMA_ERR_UNSUPPORTED, "tdma_solve_shared unavailable for this shape (see the first call)");
    }
    tdma::SharedArgs args;
    args.a_y = (const double *)a_y; args.b0_y = (const double *)b0_y; args.c_y = (const double *)c_y;
    args.sx = (const double *)sx; args.sz = (const double *)sz;
    args.d = (const double *)d; args.x = (double *)x;
    args.pin00 = pin00 ? 1 : 0;
    args.nx = pl->nx; args.ny = pl->ny; args.nzs = 0;
    args.rs = pl->rs; args.os = pl->os;
    args.axis_z = pl->axis == TDMA_AXIS_Z ? 1 : 0; args.periodic = pl->periodic ? 1 : 0;
    args.uniform = uniform ? 1 : 0;
    cudaError_t e = tdma::launch_shared(pl->sh[q], args, origin);          // prepare: attributes, grid size
    int nzf = 0;
    if (e == cudaSuccess && pl->sh_have_fill[q]) {
        e = tdma::launch_shared(pl->sh_fill[q], args, origin);
        if (e == cudaSuccess) {
            // the fill launch, as for the general kernel (enqueue_fused): clusters of 2 on the SMs
            // the main launch's clusters cannot be placed on, solving the last nzf slices
            const long per_sm = pl->sh[q].ctas_per_sm;
            const int main_ctas = pl->sh[q].max_clusters * pl->sh[q].cluster;
            const int idle = per_sm == 1 ? pl->sm_count - main_ctas : 0;
            int fc = idle / pl->sh_fill[q].cluster;
            if (fc > pl->sh_fill[q].max_clusters) fc = pl->sh_fill[q].max_clusters;
            if (fc > 0) {
                const double w = 0.8 * fc * pl->sh_fill[q].cluster;
                const double share = pl->fill_opt > 0 ? pl->fill_opt * 1e-3 : w / (w + main_ctas);
                nzf = (int)(pl->nz * share + 0.5);
                if (nzf >= pl->nz) nzf = pl->nz - 1;
                if (nzf > 0) pl->sh_fill[q].max_clusters = fc;
            }
        }
    }
    if (e != cudaSuccess) return set_err(TDMA_ERR_CUDA, "shared launch preparation failed: %s", cudaGetErrorString(e));
    pl->sh_last = q; pl->sh_fill_last = nzf;
    if (nzf > 0) {
        CUDA_TRY(cudaEventRecord(pl->evFork, origin));
        CUDA_TRY(cudaStreamWaitEvent(pl->sB, pl->evFork, 0));
    }
    args.nzs = pl->nz - nzf;
    e = tdma::launch_shared(pl->sh[q], args, origin);
    if (e == cudaSuccess && nzf > 0) {
        tdma::SharedArgs fa = args;
        const size_t off = (size_t)(pl->nz - nzf) * (size_t)pl->os * (size_t)ncomp;
        fa.d = args.d + off; fa.x = args.x + off; fa.sz = uniform ? nullptr : args.sz + (pl->nz - nzf);
        fa.pin00 = 0;                    // line (0,0) lies in slice 0, which the main launch owns
        fa.nzs = nzf;
        e = tdma::launch_shared(pl->sh_fill[q], fa, pl->sB);
        cudaError_t ej = cudaEventRecord(pl->evBJoin, pl->sB);
        if (ej == cudaSuccess) ej = cudaStreamWaitEvent(origin, pl->evBJoin, 0);
        if (e == cudaSuccess) e = ej;
    }
    if (e != cudaSuccess) return set_err(TDMA_ERR_CUDA, "shared launch failed: %s", cudaGetErrorString(e));
    return TDMA_OK;
}

int tdma_solve_host(tdma_plan *plan, const void *a, const void *b, const void *c, const void *d,
                    void *x)
{
    int rc = check_ptrs(plan, a, b, c, d, x);
    if (rc != TDMA_OK) return rc;
    tdma_plan *pl = plan;
    const bool zsw = pl->axis == TDMA_AXIS_Z;      // chunks of y-slices: strided in the caller's arrays
    if (!pl->sH2D) {  // first use: staging buffers, copy streams
        // chunk = about 16 Mi cells (128 MiB per array), or options.host_chunk slices.  PIPELINED:
        // rounded to whole batches so that the batch boundaries (and with them the bits of x) are
        // those of tdma_solve; FUSED: `batch` only chunks launches, so the target alone decides.
        const size_t target = (size_t)1 << 24;
        long long hz = pl->host_chunk > 0 ? pl->host_chunk : (long long)std::max<size_t>(1, target / pl->slice);
        if (pl->variant != TDMA_VARIANT_FUSED) hz = std::max<long long>(pl->bz, hz / pl->bz * pl->bz);
        pl->hz = (int)std::min<long long>(hz, pl->nz);
        const size_t bytes = (size_t)pl->hz * pl->slice * sizeof(double);
        if (zsw) {
            // A chunk of hz y-slices of a z sweep is a slab of its own, (nx, hz, line length), with its own
            // row stride: it gets its own plan (same options), and so does the last, shorter chunk.
            tdma_options o = pl->opt_saved;
            o.struct_size = (int)sizeof(o); o.axis = TDMA_AXIS_Z; o.periodic = pl->periodic; o.variant = pl->variant;
            const int tail = pl->nz % pl->hz;
            for (int t = 0; t < (tail ? 2 : 1); ++t) {
                const int hzc = t == 0 ? pl->hz : tail;
                const int bzc = pl->variant == TDMA_VARIANT_FUSED ? 0 : std::min(pl->bz, hzc);
                free_plan(pl->zchild[t]);
                pl->zchild[t] = tdma_plan_create_ex(pl->nx, hzc, pl->ny, pl->P, bzc, TDMA_F64, &o);
                if (!pl->zchild[t]) return g_err_code;       // message set by the failed creation
            }
        }
        for (int s = 0; s < 2; ++s)
            for (int i = 0; i < 5; ++i)
                if (cudaMalloc(&pl->stage_dev[s][i], bytes) != cudaSuccess) {
                    cudaGetLastError();
                    return set_err(TDMA_ERR_ALLOC, "cannot allocate %zu bytes of host staging", bytes);
                }
        pl->workspace += 10 * bytes;
        CUDA_TRY(cudaStreamCreateWithFlags(&pl->sH2D, cudaStreamNonBlocking));
        CUDA_TRY(cudaStreamCreateWithFlags(&pl->sD2H, cudaStreamNonBlocking));
        for (int s = 0; s < 2; ++s) {
            CUDA_TRY(cudaEventCreateWithFlags(&pl->evH2D[s], cudaEventDisableTiming));
            CUDA_TRY(cudaEventCreateWithFlags(&pl->evDone[s], cudaEventDisableTiming));
            CUDA_TRY(cudaEventCreateWithFlags(&pl->evD2H[s], cudaEventDisableTiming));
        }
    }
    const double *h[4] = {(const double *)a, (const double *)b, (const double *)c, (const double *)d};
    double *hx = (double *)x;
    const int nchunks = (pl->nz + pl->hz - 1) / pl->hz;
    for (int q = 0; q < nchunks; ++q) {
        const int s = q & 1;
        const int k0 = q * pl->hz;
        const int nzc = std::min(pl->hz, pl->nz - k0);
        const size_t off = (size_t)k0 * pl->slice;
        const size_t bytes = (size_t)nzc * pl->slice * sizeof(double);
        if (q >= 2) {  // staging slot s is free once chunk q-2 is solved and copied out
            CUDA_TRY(cudaStreamWaitEvent(pl->sH2D, pl->evDone[s], 0));
            CUDA_TRY(cudaStreamWaitEvent(pl->sH2D, pl->evD2H[s], 0));
        }
        // z sweep: rows of the line are caller z-slices, a chunk is nx * nzc contiguous doubles of each
        const size_t zoff = (size_t)k0 * pl->nx, zrow = (size_t)pl->nx * nzc * sizeof(double),
                     zpitch = (size_t)pl->nx * pl->nz * sizeof(double);
        for (int i = 0; i < 4; ++i) {
            if (zsw)
                CUDA_TRY(cudaMemcpy2DAsync(pl->stage_dev[s][i], zrow, h[i] + zoff, zpitch, zrow, (size_t)pl->ny,
                                           cudaMemcpyHostToDevice, pl->sH2D));
            else
                CUDA_TRY(cudaMemcpyAsync(pl->stage_dev[s][i], h[i] + off, bytes, cudaMemcpyHostToDevice, pl->sH2D));
        }
        CUDA_TRY(cudaEventRecord(pl->evH2D[s], pl->sH2D));
        CUDA_TRY(cudaStreamWaitEvent(pl->sMain, pl->evH2D[s], 0));
        const SlabPtrs ptr{pl->stage_dev[s][0], pl->stage_dev[s][1], pl->stage_dev[s][2],
                           pl->stage_dev[s][3], pl->stage_dev[s][4]};
        tdma_plan *solver = zsw ? pl->zchild[nzc == pl->hz ? 0 : 1] : pl;
        if ((rc = run_solve(solver, ptr, nzc, pl->sMain)) != TDMA_OK) return rc;
        CUDA_TRY(cudaEventRecord(pl->evDone[s], pl->sMain));
        CUDA_TRY(cudaStreamWaitEvent(pl->sD2H, pl->evDone[s], 0));
        if (zsw)
            CUDA_TRY(cudaMemcpy2DAsync(hx + zoff, zpitch, pl->stage_dev[s][4], zrow, zrow, (size_t)pl->ny,
                                       cudaMemcpyDeviceToHost, pl->sD2H));
        else
            CUDA_TRY(cudaMemcpyAsync(hx + off, pl->stage_dev[s][4], bytes, cudaMemcpyDeviceToHost, pl->sD2H));
        CUDA_TRY(cudaEventRecord(pl->evD2H[s], pl->sD2H));
    }
    CUDA_TRY(cudaStreamSynchronize(pl->sD2H));
    CUDA_TRY(cudaStreamSynchronize(pl->sMain));
    return TDMA_OK;
}

int tdma_plan_timeline(tdma_plan *plan, double *rec, int max_launches)
{
    if (!plan || !rec || max_launches < 0) return set_err(TDMA_ERR_INVALID_ARG, "NULL argument");
    if (!plan->timeline) return set_err(TDMA_ERR_UNSUPPORTED, "plan was not created with options.timeline = 1");
    CUDA_TRY(cudaDeviceSynchronize());
    const int n = std::min<int>((int)plan->tl_tag.size(), max_launches);
    // origin = the earliest start (launch order is not time order across streams)
    for (int i = 0; i < n; ++i) {
        float t0 = 0, t1 = 0;
        CUDA_TRY(cudaEventElapsedTime(&t0, plan->tl_ev[0], plan->tl_ev[2 * i]));
        CUDA_TRY(cudaEventElapsedTime(&t1, plan->tl_ev[0], plan->tl_ev[2 * i + 1]));
        rec[4 * i] = plan->tl_tag[i] >> 20; rec[4 * i + 1] = plan->tl_tag[i] & ((1 << 20) - 1);
        rec[4 * i + 2] = t0; rec[4 * i + 3] = t1;
    }
    return n;
}

double tdma_pipeline_model(int nb, double tA, double tB, double tC, int nstreams, double last_frac)
{
    if (nb < 1 || nstreams < 1 || nstreams > kMaxLanes + 1 || !(last_frac > 0.0) || last_frac > 1.0 ||
        tA < 0 || tB < 0 || tC < 0)
        return -1.0;
    auto dur = [&](double t, int n) { return n == nb - 1 ? t * last_frac : t; };
    if (nstreams == 1) {
        double T = 0;
        for (int n = 0; n < nb; ++n) T += dur(tA, n) + dur(tB, n) + dur(tC, n);
        return T;
    }
    // the event graph of enqueue_pipelined, stream clocks instead of launches
    const int nl = nstreams - 1, depth = nl + 2;
    std::vector<double> lane(nl, 0.0), evA(depth, 0.0), evB(depth, 0.0), evC(depth, 0.0);
    double sB = 0.0;
    for (int n = 0; n < nb + 2; ++n) {
        if (n < nb) {
            double &st = lane[n % nl];
            if (n >= depth) st = std::max(st, evC[n % depth]);
            st += dur(tA, n);
            evA[n % depth] = st;
        }
        if (n - 1 >= 0 && n - 1 < nb) {
            const int q = n - 1;
            sB = std::max(sB, evA[q % depth]) + dur(tB, q);
            evB[q % depth] = sB;
        }
        if (n - 2 >= 0 && n - 2 < nb) {
            const int q = n - 2;
            double &st = lane[q % nl];
            st = std::max(st, evB[q % depth]) + dur(tC, q);
            evC[q % depth] = st;
        }
    }
    double T = sB;
    for (double v : lane) T = std::max(T, v);
    return T;
}

int tdma_plan_autotune(int nx, int ny, int nz, int P, int dtype, int nstreams, const int *candidates,
                       int ncand, const void *a, const void *b, const void *c, const void *d, void *x,
                       int *best_batch, double *est_ms)
{
    if (!candidates || ncand < 1 || !best_batch || !a || !b || !c || !d || !x)
        return set_err(TDMA_ERR_INVALID_ARG, "NULL argument or no candidates");
    if (nstreams == 0) nstreams = 2;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    CUDA_TRY(cudaEventCreate(&e0));
    CUDA_TRY(cudaEventCreate(&e1));
    double best = -1.0;
    int rc = TDMA_OK;
    for (int i = 0; i < ncand && rc == TDMA_OK; ++i) {
        const int bz = candidates[i];
        if (est_ms) est_ms[i] = -1.0;
        if (bz < 1 || bz > nz) continue;
        const int nzs = (int)std::min<long long>(nz, 4LL * bz);          // a few batches are enough
        tdma_options opt;
        memset(&opt, 0, sizeof(opt));
        opt.struct_size = (int)sizeof(opt); opt.variant = TDMA_VARIANT_PIPELINED; opt.nstreams = nstreams;
        tdma_plan *pl = tdma_plan_create_ex(nx, ny, nzs, P, bz, dtype, &opt);
        if (!pl) { rc = TDMA_ERR_INVALID_ARG; break; }
        const int nbs = nzs / bz > 0 ? nzs / bz : 1;                     // full batches only
        double t[3] = {0, 0, 0};
        const int stages[3] = {TDMA_STAGE_A, TDMA_STAGE_B, TDMA_STAGE_C};
        for (int s = 0; s < 3 && rc == TDMA_OK; ++s) {
            for (int pass = 0; pass < 3 && rc == TDMA_OK; ++pass) {      // pass 0 warms up
                if (pass == 1) cudaEventRecord(e0, nullptr);
                for (int n = 0; n < nbs && rc == TDMA_OK; ++n)
                    rc = tdma_stage(pl, stages[s], n, a, b, c, d, x, nullptr);
            }
            cudaEventRecord(e1, nullptr);
            if (cudaEventSynchronize(e1) != cudaSuccess) rc = set_err(TDMA_ERR_CUDA, "autotune timing failed");
            float ms = 0;
            cudaEventElapsedTime(&ms, e0, e1);
            t[s] = ms / (2.0 * nbs);
        }
        tdma_plan_destroy(pl);
        if (rc != TDMA_OK) break;
        const int nb = (nz + bz - 1) / bz;
        const double last = (double)(nz - (nb - 1) * bz) / bz;
        const double est = tdma_pipeline_model(nb, t[0], t[1], t[2], nstreams, last);
        if (est_ms) est_ms[i] = est;
        if (best < 0 || est < best) { best = est; *best_batch = bz; }
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (rc == TDMA_OK && best < 0) return set_err(TDMA_ERR_INVALID_ARG, "no valid candidate batch size");
    return rc;
}

int tdma_plan_get(const tdma_plan *plan, int what)
{
    if (!plan) return set_err(TDMA_ERR_INVALID_ARG, "plan is NULL");
    switch (what) {
    case TDMA_GET_NB: return plan->nb;
    case TDMA_GET_M: return plan->m;
    case TDMA_GET_BATCH: return plan->bz;
    case TDMA_GET_NSTREAMS: return plan->variant == TDMA_VARIANT_FUSED ? 1 : plan->nstreams;
    case TDMA_GET_DEPTH: return plan->depth;
    case TDMA_GET_VARIANT: return plan->variant;
    case TDMA_GET_LAUNCHES: return launches_per_solve(plan);
    case TDMA_GET_FUSED_IMPL: return plan->fused_impl;
    case TDMA_GET_FUSED_FILL: return plan->fill_last;
    case TDMA_GET_FUSED_LINES: return plan->fused_impl == 2 ? plan->tfused.lines : plan->fused.lines;
    case TDMA_GET_FUSED_CLUSTER: return plan->fused_impl == 2 ? plan->tfused.cluster : plan->fused.cluster;
    case TDMA_GET_GRAPH_BUILDS: return plan->graph_builds;
    case TDMA_GET_FUSED_LEAF_ROWS: return plan->fused_impl == 2 ? plan->tfused.leaf_rows : plan->fused.leaf_rows;
    case TDMA_GET_FUSED_TOP: return plan->fused_impl == 2 ? 2 : plan->fused.top_mode;
    case TDMA_GET_FUSED_THREADS: return plan->fused_impl == 2 ? plan->tfused.threads : plan->fused.threads;
    case TDMA_GET_FUSED_SMEM: return (int)(plan->fused_impl == 2 ? plan->tfused.smem : plan->fused.smem);
    case TDMA_GET_FUSED_TOP_ROWS:
        return plan->fused_impl == 2 ? 2 * plan->tfused.cluster : 2 * plan->fused.top_nodes * plan->fused.cluster;
    case TDMA_GET_SHARED_LINES: return plan->sh_last < 0 ? 0 : plan->sh[plan->sh_last].lines;
    case TDMA_GET_SHARED_CLUSTER: return plan->sh_last < 0 ? 0 : plan->sh[plan->sh_last].cluster;
    case TDMA_GET_SHARED_LEAF_ROWS: return plan->sh_last < 0 ? 0 : plan->sh[plan->sh_last].leaf_rows;
    case TDMA_GET_SHARED_THREADS: return plan->sh_last < 0 ? 0 : plan->sh[plan->sh_last].threads;
    case TDMA_GET_SHARED_SMEM: return plan->sh_last < 0 ? 0 : (int)plan->sh[plan->sh_last].smem;
    case TDMA_GET_SHARED_SLOTS: return plan->sh_last < 0 ? 0 : plan->sh[plan->sh_last].slots;
    case TDMA_GET_REDUCED_PARTITIONS: return plan->Pred;
    case TDMA_GET_SHARED_LINE_KERNEL: return plan->sh_lines_last;
    case TDMA_GET_SHARED_FILL: return plan->sh_last < 0 ? 0 : plan->sh_fill_last;
    default: return set_err(TDMA_ERR_INVALID_ARG, "unknown query %d", what);
    }
}

size_t tdma_plan_workspace_bytes(const tdma_plan *plan) { return plan ? plan->workspace : 0; }

int tdma_plan_buffer(const tdma_plan *plan, int which, int slot, void **device_ptr, size_t *bytes)
{
    if (!plan || !device_ptr || !bytes) return set_err(TDMA_ERR_INVALID_ARG, "NULL argument");
    if (!plan->red || (which >= TDMA_BUF_SA && !plan->scratch))
        return set_err(TDMA_ERR_UNSUPPORTED, "plan has no such stage buffer");
    if (slot < 0 || slot >= plan->depth) return set_err(TDMA_ERR_INVALID_ARG, "slot %d outside [0, %d)", slot, plan->depth);
    switch (which) {
    case TDMA_BUF_RA: case TDMA_BUF_RC: case TDMA_BUF_RD:
        *device_ptr = slot_red(plan, slot, which - TDMA_BUF_RA);
        *bytes = (size_t)2 * plan->Pred * plan->Lb_max * sizeof(double);
        return TDMA_OK;
    case TDMA_BUF_Y:
        *device_ptr = slot_red(plan, slot, 4);
        *bytes = (size_t)2 * plan->Pred * plan->Lb_max * sizeof(double);
        return TDMA_OK;
    case TDMA_BUF_SA: case TDMA_BUF_SC: case TDMA_BUF_SD:
        *device_ptr = slot_scratch(plan, slot, which - TDMA_BUF_SA);
        *bytes = (size_t)plan->bz * plan->slice * sizeof(double);
        return TDMA_OK;
    default: return set_err(TDMA_ERR_INVALID_ARG, "unknown buffer %d", which);
    }
}

int tdma_plan_destroy(tdma_plan *plan)
{
    if (!plan) return set_err(TDMA_ERR_INVALID_ARG, "plan is NULL");
    cudaError_t e = cudaDeviceSynchronize();
    free_plan(plan);
    if (e != cudaSuccess) return set_err(TDMA_ERR_CUDA, "cudaDeviceSynchronize: %s", cudaGetErrorString(e));
    return TDMA_OK;
}

const char *tdma_last_error(void) { return g_err; }
int tdma_last_status(void) { return g_err_code; }
int tdma_version(void) { return TDMA_VERSION_NUM; }

}  // extern "C"
