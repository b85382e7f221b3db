// y-slab decomposition over several GPUs -- the paper's own setting:
// "the domain is decomposed along the y-direction" (Fig. 1c), every rank reduces its
// slab to boundary equations (stage A), an all-to-all deals the lines of a batch out evenly so that
// every rank solves a share of the reduced systems (stage B; "even distribution", PAPER.md:106,
// Alg. 2 :179-203), a second all-to-all returns the two boundary unknowns per partition and the
// ranks back-substitute (stage C).  This unit holds the rank-local stages; the exchange itself is
// the caller's: either a library all-to-all between the stages (torch.distributed
// all_to_all_single over NCCL in yslab.py), or -- tdma_slab_set_peers + the _peer entry points --
// NO separate exchange at all: stage A and stage B store every block of their output straight
// into the destination rank's receive buffer (peer memory over NVLink, or the same device), so
// the transfer overlaps the stage tile by tile and only a cross-rank barrier remains.
//
// Buffers of one batch (Lb = nx * slices lines, Ls = Lb / nranks lines per rank, P = local
// partitions per rank, Ptot = P * nranks; all doubles, line fastest):
//   send  [nranks dest][P][6][Ls]   stage A out:  (fa, fc, fd | pa, pc, pd) of partition p, i.e. rows
//                                   2p and 2p+1 of the reduced system (unit diagonal) of line
//                                   dest * Ls + j; after the all-to-all the receiver holds
//   recv  [nranks src][P][6][Ls]  = [Ptot][6][Ls]: all 2 Ptot rows of its Ls lines
//   yout  [nranks dest][2 P][Ls]  = Y[2 Ptot][Ls]  stage B out: the reduced solution, rows 2 pg, 2 pg + 1
//                                   of global partition pg = dest * P + p; after the all-to-all
//   yrecv [nranks src][2 P][Ls]     x_first / x_last of MY partitions for the lines rank src solved.
#include "../../include/tdma.h"

#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <new>

#include "tdma_stage_kernels.cuh"
#include "tdma_staged.h"

namespace {
constexpr int kU = 4;
constexpr int kSlabDepth = 3;   // batches in flight: A(n), B(n-1), C(n-2)
}

struct tdma_slab {
    int nx = 0, ny = 0, nz = 0, P = 0, m = 0, rank = 0, nranks = 0, bz = 0, nb = 0;
    long long Lb = 0, Ls = 0;
    // stage A / C: the TMA-staged kernels of the STAGED variant (nothing spilled, stage C re-reads the
    // inputs stage A was given) when the slab tiles; else the one-thread-per-(line, partition) kernels
    bool tma = false;
    tdma::StagedConfig staged;
    const double *in[kSlabDepth][4] = {};   // a, b, c, d of the batch in each ring slot (tma: for stage C)
    double *scratch = nullptr;   // depth x {a', c', d'} x [bz][ny][nx]   (not with tma)
    double *red = nullptr;       // depth x {RA, RC, RD, CP} x [2 Ptot][Ls]
    double **peer_tab = nullptr; // device: depth x {recv, yrecv} x [nranks] pointers (tdma_slab_set_peers)
    bool have_peers[kSlabDepth] = {};
    size_t workspace = 0;
};

namespace {

int slab_err(int code) { return code; }

// lines and slices of batch n (the last batch may be shorter: PAPER.md:236, 387)
bool batch_range(const tdma_slab *s, int n, int *k0, int *bzn)
{
    if (n < 0 || n >= s->nb) return false;
    *k0 = n * s->bz;
    *bzn = s->bz < s->nz - *k0 ? s->bz : s->nz - *k0;
    return true;
}

tdma::StageParams slab_params(const tdma_slab *s, int n, int k0, int bzn)
{
    tdma::StageParams prm = {};
    const int slot = n % kSlabDepth;
    const size_t per = (size_t)s->bz * s->ny * s->nx;
    prm.sa = s->scratch + ((size_t)slot * 3 + 0) * per;
    prm.sc = s->scratch + ((size_t)slot * 3 + 1) * per;
    prm.sd = s->scratch + ((size_t)slot * 3 + 2) * per;
    const int Ptot = s->P * s->nranks;
    const size_t rper = (size_t)2 * Ptot * (size_t)s->Ls;
    prm.ra = s->red + ((size_t)slot * 4 + 0) * rper;
    prm.rc = s->red + ((size_t)slot * 4 + 1) * rper;
    prm.rd = s->red + ((size_t)slot * 4 + 2) * rper;
    prm.cp = s->red + ((size_t)slot * 4 + 3) * rper;
    prm.nx = s->nx; prm.ny = s->ny; prm.m = s->m; prm.P = s->P;
    prm.rs = s->nx; prm.os = (long long)s->nx * s->ny;
    prm.Lb = (long long)s->nx * bzn;
    prm.Ls = prm.Lb / s->nranks;
    prm.pg0 = s->rank * s->P; prm.Ptot = Ptot;
    (void)k0;
    return prm;
}

}  // namespace

extern "C" {

tdma_slab *tdma_slab_create(int nx, int ny_local, int nz, int P_local, int batch, int rank, int nranks)
{
    if (nx < 1 || ny_local < 2 || nz < 1 || P_local < 1 || nranks < 1 || rank < 0 || rank >= nranks ||
        ny_local % P_local != 0 || ny_local / P_local < 2 || batch < 0 || batch > nz)
        return nullptr;
    const int bz = batch == 0 ? nz : batch;
    // even distribution of the lines of every batch (including the last, shorter one)
    if (((long long)nx * bz) % nranks != 0 || ((long long)nx * (nz % bz)) % nranks != 0) return nullptr;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return nullptr;   // no CPU fallback
    tdma_slab *s = new (std::nothrow) tdma_slab();
    if (!s) return nullptr;
    s->nx = nx; s->ny = ny_local; s->nz = nz; s->P = P_local; s->m = ny_local / P_local;
    s->rank = rank; s->nranks = nranks; s->bz = bz; s->nb = (nz + bz - 1) / bz;
    s->Lb = (long long)nx * bz; s->Ls = s->Lb / nranks;
    {
        int dev = 0;
        cudaDeviceProp prop;
        const char *why = nullptr;
        if (cudaGetDevice(&dev) == cudaSuccess && cudaGetDeviceProperties(&prop, dev) == cudaSuccess && prop.major >= 10 &&
            tdma::configure_staged(&s->staged, nx, ny_local, P_local, false, prop, &why)) {
            s->tma = true;
            s->P = s->staged.Pe;            // the exchanged level of the recursion (D1): >= 1 per CTA
            s->m = ny_local / s->P;
        }
    }
    P_local = s->P;
    const size_t sbytes = s->tma ? 0 : (size_t)kSlabDepth * 3 * bz * ny_local * nx * sizeof(double);
    const size_t rbytes = (size_t)kSlabDepth * 4 * 2 * P_local * nranks * (size_t)s->Ls * sizeof(double);
    if ((sbytes && cudaMalloc(&s->scratch, sbytes) != cudaSuccess) || cudaMalloc(&s->red, rbytes) != cudaSuccess) {
        cudaGetLastError();
        cudaFree(s->scratch); cudaFree(s->red);
        delete s;
        return nullptr;
    }
    s->workspace = sbytes + rbytes;
    return s;
}

int tdma_slab_get(const tdma_slab *s, int what)
{
    if (!s) return TDMA_ERR_INVALID_ARG;
    switch (what) {
    case TDMA_SLAB_NB: return s->nb;
    case TDMA_SLAB_BATCH: return s->bz;
    case TDMA_SLAB_LINES: return (int)s->Lb;
    case TDMA_SLAB_SHARE: return (int)s->Ls;
    case TDMA_SLAB_PTOT: return s->P * s->nranks;
    case TDMA_SLAB_PLOCAL: return s->P;
    case TDMA_SLAB_TMA: return s->tma ? 1 : 0;
    default: return TDMA_ERR_INVALID_ARG;
    }
}

int tdma_slab_set_peers(tdma_slab *s, int slot, const void *const *recv_of_rank, const void *const *yrecv_of_rank)
{
    if (!s || slot < 0 || slot >= kSlabDepth || !recv_of_rank || !yrecv_of_rank) return slab_err(TDMA_ERR_INVALID_ARG);
    for (int q = 0; q < s->nranks; ++q)
        if (!recv_of_rank[q] || !yrecv_of_rank[q] || (((uintptr_t)recv_of_rank[q] | (uintptr_t)yrecv_of_rank[q]) & 7) != 0)
            return slab_err(TDMA_ERR_INVALID_ARG);
    if (!s->peer_tab && cudaMalloc(&s->peer_tab, (size_t)kSlabDepth * 2 * s->nranks * sizeof(double *)) != cudaSuccess) {
        cudaGetLastError();
        return slab_err(TDMA_ERR_ALLOC);
    }
    double **row = s->peer_tab + (size_t)slot * 2 * s->nranks;
    // synchronous copies: the table is set up once, before the first batch
    if (cudaMemcpy(row, recv_of_rank, (size_t)s->nranks * sizeof(double *), cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(row + s->nranks, yrecv_of_rank, (size_t)s->nranks * sizeof(double *), cudaMemcpyHostToDevice) != cudaSuccess)
        return slab_err(TDMA_ERR_CUDA);
    s->have_peers[slot] = true;
    return TDMA_OK;
}

static int slab_stage_a(tdma_slab *s, int batch_index, const void *a, const void *b, const void *c,
                        const void *d, void *send, void *stream, bool peer)
{
    int k0, bzn;
    if (!s || !a || !b || !c || !d || (!send && !peer) || !batch_range(s, batch_index, &k0, &bzn)) return slab_err(TDMA_ERR_INVALID_ARG);
    if (peer && !s->have_peers[batch_index % kSlabDepth]) return slab_err(TDMA_ERR_INVALID_ARG);
    tdma::StageParams prm = slab_params(s, batch_index, k0, bzn);
    if (peer) {     // my block [src = rank] of every receiver's recv[src][P][6][Ls]
        prm.peer = s->peer_tab + (size_t)(batch_index % kSlabDepth) * 2 * s->nranks;
        prm.peer_off = (long long)s->rank * s->P * 6 * prm.Ls;
    }
    const size_t off = (size_t)k0 * (size_t)prm.os;
    prm.a = (const double *)a + off; prm.b = (const double *)b + off;
    prm.c = (const double *)c + off; prm.d = (const double *)d + off;
    prm.send = (double *)send;
    if (s->tma) {
        if ((((uintptr_t)a | (uintptr_t)b | (uintptr_t)c | (uintptr_t)d) & 15) != 0) return TDMA_ERR_UNSUPPORTED;
        const int slot = batch_index % kSlabDepth;
        s->in[slot][0] = prm.a; s->in[slot][1] = prm.b; s->in[slot][2] = prm.c; s->in[slot][3] = prm.d;
        cudaError_t e = tdma::launch_staged_slab(s->staged, 1, prm.a, prm.b, prm.c, prm.d, nullptr, prm.send, nullptr, s->nx,
                                                 s->ny, bzn, s->rank * s->ny, s->ny * s->nranks, prm.Ls, (cudaStream_t)stream,
                                                 prm.peer, prm.peer_off);
        return e == cudaSuccess ? TDMA_OK : TDMA_ERR_CUDA;
    }
    dim3 grid((unsigned)((prm.Lb + 127) / 128), s->P);
    tdma::stage_a_kernel<kU, tdma::kOutSlab><<<grid, 128, 0, (cudaStream_t)stream>>>(prm);
    return cudaGetLastError() == cudaSuccess ? TDMA_OK : TDMA_ERR_CUDA;
}

int tdma_slab_stage_a(tdma_slab *s, int batch_index, const void *a, const void *b, const void *c,
                      const void *d, void *send, void *stream)
{
    return slab_stage_a(s, batch_index, a, b, c, d, send, stream, false);
}

int tdma_slab_stage_a_peer(tdma_slab *s, int batch_index, const void *a, const void *b, const void *c,
                           const void *d, void *stream)
{
    return slab_stage_a(s, batch_index, a, b, c, d, nullptr, stream, true);
}

static int slab_stage_b(tdma_slab *s, int batch_index, const void *recv, void *yout, void *stream, bool pdd, bool peer = false)
{
    int k0, bzn;
    if (!s || !recv || (!yout && !peer) || !batch_range(s, batch_index, &k0, &bzn)) return slab_err(TDMA_ERR_INVALID_ARG);
    if (peer && !s->have_peers[batch_index % kSlabDepth]) return slab_err(TDMA_ERR_INVALID_ARG);
    tdma::StageParams prm = slab_params(s, batch_index, k0, bzn);
    if (peer) {     // my block [src = rank] of every receiver's yrecv[src][2 P][Ls]
        prm.peer = s->peer_tab + ((size_t)(batch_index % kSlabDepth) * 2 + 1) * s->nranks;
        prm.peer_off = (long long)s->rank * 2 * s->P * prm.Ls;
        prm.peer_rows = 2 * s->P;
    }
    // the reduced systems of MY share: Ls lines of 2 Ptot rows; recv is send_A[Ptot][6][Ls]
    prm.send = (double *)const_cast<void *>(recv);
    prm.y = (double *)yout;
    prm.P = prm.Ptot;
    prm.Lb = prm.Ls;
    const unsigned Ls = (unsigned)prm.Ls;
    dim3 grid((Ls + 255) / 256, prm.Ptot);
    tdma::gather_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>(prm);
    if (pdd) {
        dim3 gb((Ls + 127) / 128, prm.Ptot);
        tdma::stage_b_pdd_kernel<<<gb, 128, 0, (cudaStream_t)stream>>>(prm);
    } else {
        tdma::stage_b_kernel<kU><<<(Ls + 63) / 64, 64, 0, (cudaStream_t)stream>>>(prm);
    }
    return cudaGetLastError() == cudaSuccess ? TDMA_OK : TDMA_ERR_CUDA;
}

int tdma_slab_stage_b(tdma_slab *s, int batch_index, const void *recv, void *yout, void *stream)
{
    return slab_stage_b(s, batch_index, recv, yout, stream, false);
}

int tdma_slab_stage_b_pdd(tdma_slab *s, int batch_index, const void *recv, void *yout, void *stream)
{
    return slab_stage_b(s, batch_index, recv, yout, stream, true);
}

int tdma_slab_stage_b_peer(tdma_slab *s, int batch_index, const void *recv, int pdd, void *stream)
{
    return slab_stage_b(s, batch_index, recv, nullptr, stream, pdd != 0, true);
}

int tdma_slab_stage_c(tdma_slab *s, int batch_index, const void *yrecv, void *x, void *stream)
{
    int k0, bzn;
    if (!s || !yrecv || !x || !batch_range(s, batch_index, &k0, &bzn)) return slab_err(TDMA_ERR_INVALID_ARG);
    tdma::StageParams prm = slab_params(s, batch_index, k0, bzn);
    prm.x = (double *)x + (size_t)k0 * (size_t)prm.os;
    prm.y = (double *)const_cast<void *>(yrecv);
    if (s->tma) {
        const int slot = batch_index % kSlabDepth;
        if (!s->in[slot][0] || ((uintptr_t)x & 15) != 0) return TDMA_ERR_INVALID_ARG;     // stage A of this batch first
        cudaError_t e = tdma::launch_staged_slab(s->staged, 2, s->in[slot][0], s->in[slot][1], s->in[slot][2], s->in[slot][3],
                                                 prm.x, nullptr, prm.y, s->nx, s->ny, bzn, s->rank * s->ny,
                                                 s->ny * s->nranks, prm.Ls, (cudaStream_t)stream);
        return e == cudaSuccess ? TDMA_OK : TDMA_ERR_CUDA;
    }
    dim3 grid((unsigned)((prm.Lb + 127) / 128), s->P);
    tdma::stage_c_kernel<kU, true><<<grid, 128, 0, (cudaStream_t)stream>>>(prm);
    return cudaGetLastError() == cudaSuccess ? TDMA_OK : TDMA_ERR_CUDA;
}

int tdma_slab_destroy(tdma_slab *s)
{
    if (!s) return TDMA_ERR_INVALID_ARG;
    cudaError_t e = cudaDeviceSynchronize();
    cudaFree(s->scratch); cudaFree(s->red); cudaFree(s->peer_tab);
    if (s->staged.impl) tdma::free_staged(&s->staged);
    delete s;
    return e == cudaSuccess ? TDMA_OK : TDMA_ERR_CUDA;
}

}  // extern "C"
