// tdma_solve_static: the three-stage solve (stage A -> stage B -> stage C of PAPER.md:49-58, Alg. 1
// order) for callers that cannot allocate device memory -- code under CUDA graph
// capture, tight serving loops, harnesses that forbid cudaMalloc.  Same kernels as the PIPELINED
// variant (tdma_stage_kernels.cuh); the only difference is where the scratch lives: the modified
// coefficients a', c', d' of a batch and its reduced system sit in ONE file-scope __device__ array
// of TDMA_STATIC_SCRATCH_BYTES, which every GPU that loads the library holds until the process
// exits.  No plan, no streams or events of its own, no cudaMalloc / cudaFree / allocating library
// call anywhere on this path: the z range is cut into batches that fit the array and the batches
// run one after the other on the caller's stream.
//
// The array is SHARED by all calls and keeps the last call's contents.  Nothing in it has to
// start at zero: within a batch every element a stage reads was written earlier in the same batch
// (stage A writes all of a', c', d' and RA / RC / RD, stage B writes CP and Y before reading them),
// so stale contents are never observed and nothing is cleared.  Two calls that overlap on the GPU
// (different streams, or graph branches without a dependency) RACE on it.
#include "../../include/tdma.h"

#include <cuda_runtime.h>

#include <atomic>
#include <cstdint>
#include <cstdio>

#include "tdma_stage_kernels.cuh"

namespace tdma {
int report_error(int code, const char *msg);   // tdma_plan.cu: the message tdma_last_error() returns
}

namespace {

constexpr int kU = 4;                 // rows prefetched per step, as in the PIPELINED plan
constexpr size_t kScratchDoubles = (size_t)TDMA_STATIC_SCRATCH_BYTES / sizeof(double);
constexpr size_t kAlignDoubles = 32;  // every sub-array starts on a 256-byte boundary

// In HOST code this name is a host-side stand-in, not a device address: the kernels are given the
// pointer cudaGetSymbolAddress returns for the CURRENT device (scratch_of_current_device below).
static __device__ __align__(256) double g_static_scratch[kScratchDoubles];

constexpr int kMaxDevices = 64;
std::atomic<double *> g_scratch_addr[kMaxDevices];   // per device; nullptr = not resolved yet

size_t round_up(size_t n) { return (n + kAlignDoubles - 1) / kAlignDoubles * kAlignDoubles; }

int fail(int code, const char *fmt, long long v0 = 0, long long v1 = 0, long long v2 = 0)
{
    char msg[400];
    snprintf(msg, sizeof(msg), fmt, v0, v1, v2);
    return tdma::report_error(code, msg);
}

// Device address of the array on the current device, resolved once per device with that device
// current (the address differs from device to device).  Benign race: two threads resolving the
// same device store the same value.
int scratch_of_current_device(double **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) {
        char msg[200];
        snprintf(msg, sizeof(msg), "tdma_solve_static: cudaGetDevice failed: %s", cudaGetErrorString(e));
        return tdma::report_error(TDMA_ERR_CUDA, msg);
    }
    if (dev < 0 || dev >= kMaxDevices)
        return fail(TDMA_ERR_UNSUPPORTED, "tdma_solve_static: device index %lld outside [0, %lld)", dev, kMaxDevices);
    double *p = g_scratch_addr[dev].load(std::memory_order_acquire);
    if (!p) {
        void *sym = nullptr;
        e = cudaGetSymbolAddress(&sym, g_static_scratch);
        if (e != cudaSuccess || !sym) {
            char msg[200];
            snprintf(msg, sizeof(msg), "tdma_solve_static: cudaGetSymbolAddress failed: %s", cudaGetErrorString(e));
            return tdma::report_error(TDMA_ERR_CUDA, msg);
        }
        p = static_cast<double *>(sym);
        g_scratch_addr[dev].store(p, std::memory_order_release);
    }
    *out = p;
    return TDMA_OK;
}

// doubles of scratch a batch of bz slices needs: 3 arrays [bz][ny][nx] + 5 arrays [2P][nx * bz]
size_t batch_doubles(int nx, int ny, int P, long long bz)
{
    return 3 * round_up((size_t)nx * ny * bz) + 5 * round_up((size_t)2 * P * nx * bz);
}

}  // namespace

extern "C" int tdma_solve_static(int nx, int ny, int nz, int P, const void *a, const void *b, const void *c,
                                 const void *d, void *x, void *stream)
{
    if (nx < 1 || ny < 2 || nz < 1 || P < 1 || ny % P != 0 || ny / P < 2)
        return fail(TDMA_ERR_INVALID_ARG, "tdma_solve_static: needs nx, nz >= 1, P >= 1 dividing ny, ny / P >= 2 (ny = %lld, P = %lld)", ny, P);
    if (P > 65535) return fail(TDMA_ERR_UNSUPPORTED, "tdma_solve_static: P = %lld exceeds 65535", P);
    if (!a || !b || !c || !d || !x) return fail(TDMA_ERR_INVALID_ARG, "tdma_solve_static: NULL array");
    if ((((uintptr_t)a | (uintptr_t)b | (uintptr_t)c | (uintptr_t)d | (uintptr_t)x) & 7) != 0)
        return fail(TDMA_ERR_INVALID_ARG, "tdma_solve_static: arrays must be 8-byte aligned");
    // the largest batch of z-slices whose a', c', d' and reduced system fit the static array
    const size_t one = batch_doubles(nx, ny, P, 1);
    if (one > kScratchDoubles)
        return fail(TDMA_ERR_UNSUPPORTED,
                    "tdma_solve_static: one z-slice of this shape needs %lld bytes of scratch, the static array holds "
                    "%lld (TDMA_STATIC_SCRATCH_BYTES); use a plan (tdma_plan_create / tdma_solve)",
                    (long long)(one * sizeof(double)), (long long)TDMA_STATIC_SCRATCH_BYTES);
    long long bz = (long long)(kScratchDoubles / one);
    if (bz > nz) bz = nz;
    while (bz > 1 && batch_doubles(nx, ny, P, bz) > kScratchDoubles) --bz;   // rounding of the sub-arrays
    if ((long long)nx * bz > 0x7fffffffLL / 2) bz = 0x7fffffffLL / 2 / nx;     // line index fits the grid arithmetic

    double *base = nullptr;
    const int rc = scratch_of_current_device(&base);
    if (rc != TDMA_OK) return rc;

    const cudaStream_t st = (cudaStream_t)stream;
    const size_t slice = (size_t)nx * ny;
    for (long long k0 = 0; k0 < nz; k0 += bz) {
        const long long bzn = bz < nz - k0 ? bz : nz - k0;
        const size_t S = round_up(slice * (size_t)bzn), Rr = round_up((size_t)2 * P * nx * (size_t)bzn);
        tdma::StageParams prm;
        const size_t off = (size_t)k0 * slice;
        prm.a = (const double *)a + off; prm.b = (const double *)b + off;
        prm.c = (const double *)c + off; prm.d = (const double *)d + off;
        prm.x = (double *)x + off;
        prm.sa = base; prm.sc = base + S; prm.sd = base + 2 * S;
        double *red = base + 3 * S;
        prm.ra = red; prm.rc = red + Rr; prm.rd = red + 2 * Rr; prm.cp = red + 3 * Rr; prm.y = red + 4 * Rr;
        prm.send = nullptr;
        prm.Lb = (long long)nx * bzn;
        prm.nx = nx; prm.ny = ny; prm.m = ny / P; prm.P = P;
        prm.rs = nx; prm.os = (long long)slice;
        prm.pg0 = 0; prm.Ptot = P; prm.Ls = 0;
        const unsigned Lb = (unsigned)prm.Lb;
        const dim3 grid((Lb + 127) / 128, (unsigned)P);
        tdma::stage_a_kernel<kU, tdma::kOutReduced><<<grid, 128, 0, st>>>(prm);
        tdma::stage_b_kernel<kU><<<(Lb + 63) / 64, 64, 0, st>>>(prm);
        tdma::stage_c_kernel<kU, false><<<grid, 128, 0, st>>>(prm);
        const cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) {
            char msg[200];
            snprintf(msg, sizeof(msg), "tdma_solve_static: launch failed: %s", cudaGetErrorString(e));
            return tdma::report_error(TDMA_ERR_CUDA, msg);
        }
    }
    return TDMA_OK;
}
