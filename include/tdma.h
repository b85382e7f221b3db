/*
 * tdma.h -- C ABI of the B200-native Pipelined-TDMA hot path (arxiv 2509.03933).
 *
 * One thing is solved: for every (i,k) line of an nx*ny*nz fp64 slab, the tridiagonal system
 *
 *        a_j x_{j-1} + b_j x_j + c_j x_{j+1} = d_j ,     j = 0 .. ny-1
 *
 * ("Problem: Ax = d (N times); Input a, b, c, d; Output x", PAPER.md:127-131 / Alg. 1 and
 * PAPER.md:169-173 / Alg. 2; a, b, c = sub-, main, super-diagonal), with the
 * systems aligned with y (Fig. 1c) and the y direction split into P partitions
 * (the paper's processors p).
 *
 * LAYOUT.  Every array holds nx*ny*nz doubles, element (i,j,k) at  i + nx*(j + ny*k)  (x fastest,
 * then y, then z).  a at j = 0 and c at j = ny-1 are IGNORED (treated as 0); they need not be
 * valid numbers.  A batch is a contiguous range of z-slices.
 *
 * OWNERSHIP.  a, b, c, d, x are caller-owned.  For tdma_solve / tdma_stage they are DEVICE
 * pointers, for tdma_solve_host they are HOST pointers (pinned memory recommended).  Inputs are
 * never written.  x may alias d exactly (in place); any other overlap is undefined.  The plan
 * owns its scratch ring, reduced-system buffers, streams, events and CUDA graphs.
 *
 * ASYNCHRONY.  tdma_solve only enqueues work: it forks the plan's internal streams from `stream`
 * and joins them back, so work enqueued later on `stream` sees x.  No host synchronisation
 * inside.  One solve in flight per plan; concurrent solves need separate plans.
 *
 * ALSO HERE, each documented at its declaration: tdma_solve_shared (1-D coefficient arrays, real or
 * complex right-hand sides: the form the paper benchmarks), the tdma_slab_* calls (rank-local stages
 * of the multi-GPU y-slab decomposition, with buffered output or storing straight into the peers'
 * receive buffers), stage-isolated launches, the batch-size optimiser, the
 * stream timeline, an allocation-free solve (tdma_solve_static) and an fp64 ALU probe.
 *
 * ERRORS.  tdma_plan_create* return NULL on failure; the int-returning calls return TDMA_OK (0)
 * or a negative tdma_status; a message for the calling thread is in tdma_last_error().
 * There is no CPU fallback: without a CUDA device every compute call fails with TDMA_ERR_CUDA.
 */
#ifndef TDMA_H_
#define TDMA_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tdma_plan tdma_plan; /* opaque, library-owned */

typedef enum tdma_dtype {
    TDMA_F64 = 0 /* the only arithmetic type of the path (BASELINE.json: fp64) */
} tdma_dtype;

typedef enum tdma_status {
    TDMA_OK = 0,
    TDMA_ERR_INVALID_ARG = -1,
    TDMA_ERR_UNSUPPORTED = -2,
    TDMA_ERR_ALLOC = -3,
    TDMA_ERR_CUDA = -4
} tdma_status;

/* How the three compute stages of the divide-and-conquer solve (Fig. 5) are
 * mapped onto the GPU. */
typedef enum tdma_variant {
    /* The fastest variant that can run the plan: FUSED (TMA kernel, `batch` ignored: persistent
     * launches of about 2^27 cells each) when the shape tiles, else PIPELINED.  This is what
     * tdma_plan_create uses. */
    TDMA_VARIANT_AUTO = 0,
    /* Stage A (partition reduce, fused gather) / Stage B (reduced 2P-row solve) / Stage C
     * (back-substitution) as separate kernels, z-batches pipelined over CUDA streams with events
     * exactly as Alg. 2: A(n) || B(n-1) || C(n-2).  The partition results
     * travel A -> C through a plan-owned scratch ring in HBM/L2. */
    TDMA_VARIANT_PIPELINED = 1,
    /* One persistent kernel: a thread-block cluster owns whole lines, the partitions of a line
     * live in the shared memory of the cluster's CTAs (the paper's ranks), the reduced system is
     * exchanged through distributed shared memory (the paper's MPI_Alltoall) and
     * solved inside the cluster, so HBM sees a, b, c, d once and x once (40 B/cell).  `batch` only
     * chunks the z range into launches (0 = about 2^27 cells per launch). */
    TDMA_VARIANT_FUSED = 2,
    /* The paper's three stages as separate kernels on the Alg. 2 stream pipeline, like PIPELINED,
     * but stage A and stage C fetch their partition segments by TMA into shared memory and keep
     * the modified coefficients a', c', d' ON CHIP (north_star): stage A writes
     * only the partitions' boundary equations (reads 32 B/cell), stage C fetches the segment
     * again, re-reduces it and back-substitutes with the boundary unknowns stage B computed
     * (reads 32, writes 8 B/cell).  72 B/cell instead of PIPELINED's 88, no scratch ring.  The
     * exchanged level of the recursion is the highest whose nodes are no longer than ny/P rows
     * (TDMA_GET_REDUCED_PARTITIONS of them per line; D1).  y / z sweeps, plain or cyclic lines,
     * 16-byte aligned arrays, shapes the TMA kernel tiles. */
    TDMA_VARIANT_STAGED = 3
} tdma_variant;

/* Optional tuning knobs for tdma_plan_create_ex.  Zero-initialise, set struct_size =
 * sizeof(tdma_options); every field set to 0 means "library default". */
typedef struct tdma_options {
    int struct_size;
    int variant;         /* tdma_variant */
    int nstreams;        /* PIPELINED: 1 = sequential Alg. 1 order on one stream; 2 = {A+C, B}
                            (paper); 3..8 = (nstreams-1) A+C lanes + 1 B stream.
                            default 2 */
    int use_graph;       /* 1 = capture the schedule once per pointer set into a CUDA graph
                            (default), -1 = plain stream launches */
    int separate_gather; /* 1 = stage A writes a send_A buffer and a separate gather kernel
                            assembles the reduced system (the paper's A2B);
                            default 0 = gather fused into stage A's epilogue */
    int fused_lines;     /* FUSED: lines (x extent) per cluster tile (8, 16, 32), 0 = auto */
    int fused_cluster;   /* FUSED: CTAs per cluster (1, 2, 4, 8, 16; x sweeps also 3, 5, 6), 0 = auto */
    int fused_leaf_rows; /* FUSED: rows per thread-level leaf (a divisor of ny/P, >= 2), 0 = auto */
    int fused_top;       /* FUSED: 1 = the cluster exchanges / solves the 2P-row reduced system as
                            is; 2 = every CTA first reduces its 2P/cluster rows to two (same
                            recursion), the cluster solves 2*cluster rows; 0 = auto */
    int fused_impl;      /* FUSED: 1 = register-staged kernel with a general fan-in tree (any nx,
                            any divisor leaf); 2 = TMA kernel (tile fetched by bulk tensor copies,
                            reduced in place, pairwise tree; needs even nx and power-of-two
                            leaf counts); 0 = auto (2 when eligible, else 1) */
    int fused_fill;      /* FUSED, TMA kernel: clusters of 4 or more CTAs cannot be placed on every
                            SM (a GPC holds 16-20 SMs); 0 = auto: a second, concurrent launch with
                            clusters of 2 solves the last z-slices on the SMs the main launch
                            leaves empty; N > 0: give it N/1000 of the slices; -1 = off */
    int axis;            /* direction of the systems (BASELINE cfg 4): TDMA_AXIS_Y = 0
                            (default; lines along y, y split into P partitions, `batch` counts
                            z-slices) or TDMA_AXIS_Z = 2 (lines along z, stride nx*ny, z split into
                            P partitions, `batch` counts y-slices) or TDMA_AXIS_X = 1 (lines along
                            x, the contiguous axis, x split into P partitions, `batch` counts
                            z-slices; FUSED TMA kernel: nx a multiple of 16, 16-byte aligned
                            arrays including x; PIPELINED: any nx, with strided accesses -- the
                            fallback AUTO takes when the TMA kernel cannot tile the lines) */
    int periodic;        /* 1 = cyclic lines: row 0 couples to row n-1 through a_0 and row n-1 to
                            row 0 through c_{n-1} (both entries are then USED).  The wrap is
                            resolved at the top of the recursion: at the root of the tree in the
                            FUSED TMA kernel, in stage B's reduced system (then a cyclic 2P-row
                            system) in the PIPELINED variant, which takes any nx and line length
                            along x, y or z, and in STAGED.  AUTO picks FUSED when the shape tiles,
                            else PIPELINED; pdd and the register-staged fused kernel do plain lines only */
    int timeline;        /* PIPELINED, 1 = record a timing event before and after every stage launch
                            (forces plain stream launches); read back with tdma_plan_timeline */
    int fused_slots;     /* FUSED, TMA kernel: ring slots of one raw array tile each: 4 = the next tile is
                            fetched after the sweep of this one, 5 .. 8 = that many minus 4 arrays of the
                            next tile stay in flight during the sweep; 0 = auto (as many as shared
                            memory holds, at most 8) */
    int host_chunk;      /* tdma_solve_host: z-slices per host chunk (0 = auto, about 16 Mi cells;
                            PIPELINED plans round it to whole batches) */
    int shared_lines;    /* tdma_solve_shared: cells along x per tile (real: 16 or 32, complex: 8 or 16),
                            0 = auto (128-byte row segments) */
    int shared_cluster;  /* tdma_solve_shared: CTAs per cluster (1, 2, 4, 8; x sweeps also 3, 5, 6), 0 = auto */
    int shared_leaf_rows;/* tdma_solve_shared: rows per thread-level leaf (4, 8, 16, 32; 10, 12, 20, 24), 0 = auto */
    int shared_slots;    /* tdma_solve_shared: tiles in the shared-memory ring (2 .. 4), 0 = auto */
    int pdd;             /* PIPELINED / STAGED: 1 = stage B is the Parallel Diagonally Dominant variant
                            (Sun 1995): the far ends of the partitions' spikes are
                            dropped, which leaves one 2 x 2 system per partition interface instead of
                            the 2P-row chain.  An APPROXIMATION: exact when partitions do not couple,
                            error of the order of the dropped entries otherwise (they decay
                            geometrically with ny/P for strictly dominant systems, e.g. below 1e-11
                            for the ADI sweeps of BASELINE cfg 4 with alpha <= 1 at 64 rows per partition) */
    int shared_ctas;     /* tdma_solve_shared: CTAs per SM: 1, or 2 (the <= 128-register build of the
                            16-row-leaf kernel, two CTAs co-resident); 0 = auto */
} tdma_options;

enum { TDMA_AXIS_Y = 0, TDMA_AXIS_X = 1, TDMA_AXIS_Z = 2 };

/* Plan for an nx*ny*nz slab with y split into P partitions of ny/P rows and `batch` z-slices per
 * pipeline stage (batch_z of PAPER.md:236; 0 = all slices in one batch; a last smaller batch is
 * created when nz % batch != 0).
 * Invalid: any dimension < 1, P < 1, ny % P != 0, ny/P < 2 when P > 1, batch < 0 or > nz,
 * dtype != TDMA_F64.  Returns NULL and sets tdma_last_error() on failure. */
tdma_plan *tdma_plan_create(int nx, int ny, int nz, int P, int batch, int dtype);
tdma_plan *tdma_plan_create_ex(int nx, int ny, int nz, int P, int batch, int dtype,
                               const tdma_options *options /* may be NULL */);

/* Solve all nx*nz systems.  a, b, c, d, x: DEVICE pointers to nx*ny*nz doubles (layout above).
 * stream: a cudaStream_t passed as void* (NULL = the legacy default stream).
 * Enqueue-only; returns TDMA_OK or a negative status. */
int tdma_solve(tdma_plan *plan, const void *a, const void *b, const void *c, const void *d,
               void *x, void *stream);

/* Shared-coefficient / complex right-hand-side solve -- the paper's own
 * benchmark configuration: "3D complex-valued data", a coefficient matrix
 * that "depends solely on grid spacing", shared by all systems, with the
 * FFT-reduced Poisson operator (d2/dy2 - k_l - k_m) Phi = Q.  Line (i,k) solves
 *
 *     a_y[j] x_{j-1} + (b0_y[j] - (sx[i] + sz[k])) x_j + c_y[j] x_{j+1} = d_j ,   j = 0 .. ny-1,
 *
 * the shift s = sx[i] + sz[k] being formed in fp64 before it is subtracted from b0_y[j].
 * a_y, b0_y, c_y: DEVICE pointers to ny doubles (a_y[0], c_y[ny-1] ignored); sx: nx doubles; sz: nz
 * doubles.  ncomp = 1: d, x hold nx*ny*nz doubles (layout above); ncomp = 2: complex cells,
 * interleaved (re, im), component q of cell (i,j,k) at q + 2*(i + nx*(j + ny*k)); the matrix is
 * real, so re and im are two right-hand sides of the same system.  pin00 != 0: row 0 of line
 * (0,0) is replaced by b = 1, c = 0 (the singular mean mode of the Poisson problem pinned to
 * x_0 = d_0, BASELINE cfg 2/3).  d, x: DEVICE pointers, 16-byte aligned; x may alias d exactly.
 * HBM traffic: d read once, x written once (16 B per real cell, 32 B per complex cell); the
 * matrix is rebuilt on chip.  The plan gives the shape and the sweep: lines along y, or along z
 * (options.axis = TDMA_AXIS_Z: a_y, b0_y, c_y then hold nz entries along z, sz holds ny shifts, one
 * per y-slice) -- the momentum sweeps of the paper's ADI scheme share their matrix in the same way
 * -- or along x (options.axis = TDMA_AXIS_X, ncomp = 1 only, nx a multiple of 16:
 * a_y, b0_y, c_y hold nx entries along x, sx holds NY shifts, one per line of a slice, sz the nz
 * shifts of the slices: line (j,k) has the shift sx[j] + sz[k]) -- plain or cyclic
 * (options.periodic, without pin00).
 * UNIFORM MATRIX: sx = sz = NULL (both) means every line has the same matrix a_y, b0_y, c_y -- the
 * ADI momentum sweeps, "all systems in the batch share the same matrix A"; pin00 must
 * be 0.  For real cells on shapes a 16-line tile with 16- or 32-row leaves covers, everything that
 * depends on the matrix alone (every reciprocal below the tree) is then computed once per launch
 * instead of once per line (x agrees with zero shift arrays to rounding); other shapes and complex
 * cells run the general form with plan-owned zero shifts (allocated at the first such call).
 * P and batch are not used: the line is cut into the kernel's own leaves (D1); one
 * persistent launch (plus the fill launch, see fused_fill) per call.
 * GENERAL SHAPES.  The tiled kernel needs ny = CL * W * M0 (CL in 1,2,4,8, W a power of two <= 32, M0 in
 * 4,8,16,32 or, for 3 * 2^k and 5 * 2^k lengths, 12,24 / 10,20), an even nx*ncomp, real cells for x sweeps and 16-byte aligned d, x.  Everything else (any
 * ny >= 1, odd nx, complex cells along x, 8-byte aligned arrays) runs a one-thread-per-line Thomas kernel
 * with the matrix rebuilt on the fly: correct for every shape, not fast (48 instead of 16 B per real cell:
 * c' travels through a plan-owned scratch array of at most 256 MiB, allocated at the first such call, and
 * d' through x; x sweeps strided) -- unless a tiling was requested through the shared_* options, in which
 * case the call fails with TDMA_ERR_UNSUPPORTED.  TDMA_GET_SHARED_LINE_KERNEL tells which one ran.
 * Enqueue-only. */
int tdma_solve_shared(tdma_plan *plan, const void *a_y, const void *b0_y, const void *c_y,
                      const void *sx, const void *sz, int ncomp, int pin00, const void *d, void *x,
                      void *stream);

/* Same solve with HOST buffers: the slab is streamed through plan-owned device staging buffers
 * in z-chunks (H2D copy of chunk n+1 and D2H copy of chunk n-1 overlap the solve of chunk n); a z
 * sweep is streamed in chunks of y-slices (strided 2-D copies; every chunk is a slab of its own and
 * runs on a plan of its own, created with the same options at the first call).
 * Blocks until x is complete on the host.  Pinned host memory gives asynchronous copies;
 * pageable memory works but serialises. */
int tdma_solve_host(tdma_plan *plan, const void *a, const void *b, const void *c, const void *d,
                    void *x);

/* Run ONE stage of ONE batch on `stream` (stage-isolated timing as in PAPER.md:415 "each stage
 * was timed independently", and stage-level tests).  PIPELINED plans only.  Pointers are the
 * slab base pointers as for tdma_solve; the batch's z-range is derived from batch_index.
 * Ring slot used: batch_index % TDMA_GET_DEPTH. */
typedef enum tdma_stage_id {
    TDMA_STAGE_A = 0,      /* partition reduce (+ fused gather unless separate_gather) */
    TDMA_STAGE_GATHER = 1, /* separate gather kernel (separate_gather plans only)      */
    TDMA_STAGE_B = 2,      /* reduced 2P-row solve                                      */
    TDMA_STAGE_C = 3       /* back-substitution                                         */
} tdma_stage_id;
int tdma_stage(tdma_plan *plan, int stage, int batch_index, const void *a, const void *b,
               const void *c, const void *d, void *x, void *stream);

/* Introspection. */
typedef enum tdma_query {
    TDMA_GET_NB = 0,       /* number of batches, ceil(nz / batch)                   */
    TDMA_GET_M = 1,        /* rows per partition, ny / P                            */
    TDMA_GET_BATCH = 2,    /* effective z-slices per batch                          */
    TDMA_GET_NSTREAMS = 3, /* internal streams used                                 */
    TDMA_GET_DEPTH = 4,    /* scratch ring depth (batches in flight)                */
    TDMA_GET_VARIANT = 5,  /* resolved tdma_variant                                 */
    TDMA_GET_LAUNCHES = 6, /* kernel launches one tdma_solve enqueues               */
    TDMA_GET_FUSED_LINES = 7,
    TDMA_GET_FUSED_CLUSTER = 8,
    TDMA_GET_GRAPH_BUILDS = 9, /* CUDA graphs captured so far (cache misses)       */
    TDMA_GET_FUSED_LEAF_ROWS = 10, /* rows per thread-level leaf                    */
    TDMA_GET_FUSED_TOP = 11,       /* resolved fused_top                            */
    TDMA_GET_FUSED_THREADS = 12,   /* threads per CTA                               */
    TDMA_GET_FUSED_SMEM = 13,      /* dynamic shared memory per CTA, bytes          */
    TDMA_GET_FUSED_TOP_ROWS = 14,  /* rows of the cluster-level system per line     */
    TDMA_GET_FUSED_IMPL = 15,      /* resolved fused_impl                           */
    TDMA_GET_FUSED_FILL = 16,      /* z-slices of the last solve given to the fill launch */
    /* tiling of the last tdma_solve_shared (0 before the first one) */
    TDMA_GET_SHARED_LINES = 17, TDMA_GET_SHARED_CLUSTER = 18, TDMA_GET_SHARED_LEAF_ROWS = 19,
    TDMA_GET_SHARED_THREADS = 20, TDMA_GET_SHARED_SMEM = 21, TDMA_GET_SHARED_SLOTS = 22,
    TDMA_GET_SHARED_FILL = 23,     /* z-slices its fill launch took */
    TDMA_GET_REDUCED_PARTITIONS = 24, /* partitions per line in the reduced buffers (P; STAGED: see there) */
    TDMA_GET_SHARED_LINE_KERNEL = 25  /* 1: the last tdma_solve_shared ran the one-thread-per-line kernel (a shape or
                                         alignment the tiled kernel does not take; TDMA_GET_SHARED_* are then 0) */
} tdma_query;
int tdma_plan_get(const tdma_plan *plan, int what); /* < 0 on error */
size_t tdma_plan_workspace_bytes(const tdma_plan *plan); /* device bytes the plan owns */

/* Device pointer + size of a plan-owned buffer of ring slot `slot` (tests only; PIPELINED, and the
 * reduced-system buffers of STAGED with P = TDMA_GET_REDUCED_PARTITIONS).
 * Reduced-system buffers are [2P][Lb] doubles, line fastest (Lb = nx * batch lines), unit
 * diagonal implicit; row 2p is partition p's first-row equation, row 2p+1 its last-row
 * equation.  Scratch buffers have the slab layout restricted to the batch. */
typedef enum tdma_buffer_id {
    TDMA_BUF_RA = 0, TDMA_BUF_RC = 1, TDMA_BUF_RD = 2, TDMA_BUF_Y = 3,
    TDMA_BUF_SA = 4, TDMA_BUF_SC = 5, TDMA_BUF_SD = 6
} tdma_buffer_id;
int tdma_plan_buffer(const tdma_plan *plan, int which, int slot, void **device_ptr, size_t *bytes);

/* Batch-size optimiser of the paper (sections 4.2-4.2.3), PIPELINED variant.
 *
 * tdma_pipeline_model: the "simplified pipelining structure" (Fig. 6b) as a pure host
 * function: makespan of Alg. 2's schedule (A(n) and C(n-2) on the A+C lanes, B(n-1) on its own
 * stream, event dependencies A(n) -> B(n) -> C(n), ring of nstreams+1 scratch slots) for nb batches
 * whose stages take tA, tB, tC when run alone and overlap perfectly across streams; the last batch
 * is scaled by last_frac in (0, 1] (remainder batch).  nstreams as in tdma_options
 * (1 = sequential Alg. 1 order).  Returns the time in the unit of tA/tB/tC, < 0 on bad arguments.
 *
 * tdma_plan_autotune: for every candidate batch size, times the three stages separately on the
 * first few batches of the caller's slab (mean per batch, "each stage timed independently",
 * PAPER.md:415), evaluates the model for all nz slices and returns the argmin in *best_batch and
 * the estimates (ms) in est_ms[0..ncand).  a, b, c, d, x: DEVICE pointers as for tdma_solve; x is
 * used as scratch.  Synchronises the device; not for use inside a timed region. */
/* Stream-overlap timeline of the LAST tdma_solve of a plan created with options.timeline = 1
 * (S6 evidence where nsys is not available): for launch i, rec[4i..4i+3] = stage (tdma_stage_id),
 * batch index, start and end in ms relative to the first launch of the solve, measured with CUDA
 * events on the stream the stage ran on.  Synchronises.  Returns the number of launches written
 * (<= max_launches) or a negative status. */
int tdma_plan_timeline(tdma_plan *plan, double *rec, int max_launches);

double tdma_pipeline_model(int nb, double tA, double tB, double tC, int nstreams, double last_frac);
int tdma_plan_autotune(int nx, int ny, int nz, int P, int dtype, int nstreams, const int *candidates,
                       int ncand, const void *a, const void *b, const void *c, const void *d, void *x,
                       int *best_batch, double *est_ms);

/* ---------------------------------------------------------------------------------------------
 * y-slab decomposition over several GPUs -- the paper's own multi-GPU
 * setting: "the domain is decomposed along the y-direction" (Fig. 1c); rank r owns
 * rows r*ny_local .. (r+1)*ny_local-1 of every line.  Per batch (Alg. 2):
 *   stage A  every rank reduces its slab (P_local partitions of ny_local / P_local rows) to two
 *            boundary equations per partition and writes them, 6 doubles each, into `send`;
 *   A2B      all-to-all: the Lb = nx * slices lines of the batch are dealt out evenly, Ls = Lb /
 *            nranks to each rank ("even distribution");
 *   stage B  every rank solves the 2 * P_local * nranks-row reduced systems of its Ls lines;
 *   B2C      all-to-all back: the two boundary unknowns of every partition;
 *   stage C  every rank back-substitutes inside its partitions.
 * This library provides the rank-local stages; the two all-to-alls are the caller's (yslab.py:
 * torch.distributed all_to_all_single over NCCL on a communication stream, pipelined over batches
 * as Alg. 2).  Buffer layouts (doubles, line fastest), P = P_local:
 *   send  [nranks dest][P][6][Ls]  (fa, fc, fd | pa, pc, pd): reduced rows 2p, 2p+1 (unit diagonal) of
 *                                  line dest*Ls + j;   recv = the same as [nranks src][P][6][Ls]
 *   yout  [nranks dest][2P][Ls]    reduced solution rows of rank dest's partitions for MY Ls lines;
 *   yrecv [nranks src][2P][Ls]     x_first / x_last of MY partitions for the lines rank src solved.
 * Ls is that of the batch (the last batch of nz % batch slices is shorter).  a, b, c, d, x: DEVICE
 * pointers to the rank's slab, nx*ny_local*nz doubles, element (i,j,k) at i + nx*(j + ny_local*k);
 * a at the global row 0 (rank 0) and c at the global last row (rank nranks-1) are ignored.
 * When the slab tiles for the TMA kernel (even nx, 16-byte aligned arrays, ny_local = CTAs x 2^k
 * leaves), stage A and stage C are the TMA-staged kernels of TDMA_VARIANT_STAGED: nothing is spilled,
 * stage C fetches a, b, c, d of the batch AGAIN (the pointers stage A of that batch was given: they
 * must still be valid and unchanged), and the exchanged level of the recursion -- P in the layouts
 * above -- is tdma_slab_get(TDMA_SLAB_PLOCAL), which may differ from the P_local asked for
 * (D1).  Otherwise the one-thread-per-(line, partition) kernels of PIPELINED are used.
 * Either way the slab keeps a ring of 3 batches: stage C of batch n must be enqueued before stage A
 * of batch n + 3 (Alg. 2's order A(n), B(n-1), C(n-2) does that).
 * tdma_slab_create returns NULL on invalid arguments (ny_local % P_local != 0, fewer than 2 rows per
 * partition, nx*batch or nx*(nz % batch) not divisible by nranks), without a CUDA device, or when
 * the scratch ring (3 batches of a', c', d' + reduced buffers) cannot be allocated.  Enqueue-only. */
typedef struct tdma_slab tdma_slab;
typedef enum tdma_slab_query {
    TDMA_SLAB_NB = 0, TDMA_SLAB_BATCH = 1, TDMA_SLAB_LINES = 2 /* Lb of a full batch */,
    TDMA_SLAB_SHARE = 3 /* Ls of a full batch */, TDMA_SLAB_PTOT = 4,
    TDMA_SLAB_PLOCAL = 5 /* partitions per rank actually exchanged: size the buffers with THIS P */,
    TDMA_SLAB_TMA = 6    /* 1: stage A / C are the TMA-staged kernels (72 B/cell, no scratch ring) */
} tdma_slab_query;
tdma_slab *tdma_slab_create(int nx, int ny_local, int nz, int P_local, int batch, int rank, int nranks);
int tdma_slab_get(const tdma_slab *slab, int what);
int tdma_slab_stage_a(tdma_slab *slab, int batch_index, const void *a, const void *b, const void *c,
                      const void *d, void *send, void *stream);
int tdma_slab_stage_b(tdma_slab *slab, int batch_index, const void *recv, void *yout, void *stream);
/* the same with the PDD reduced solve (tdma_options.pdd): independent 2 x 2 interface systems */
int tdma_slab_stage_b_pdd(tdma_slab *slab, int batch_index, const void *recv, void *yout, void *stream);
int tdma_slab_stage_c(tdma_slab *slab, int batch_index, const void *yrecv, void *x, void *stream);
/* Stages fused with their all-to-all: instead of filling a send / yout buffer that a
 * collective then redistributes, the kernels store block `dest` of it straight into rank dest's
 * receive buffer -- peer memory mapped into this process (NVLink P2P / symmetric memory), or any
 * device pointer -- at the place the all-to-all would have put it: block [src = rank] of
 * recv[src][P][6][Ls] / yrecv[src][2P][Ls].  The transfer then overlaps the stage tile by tile; what is
 * left of the exchange is ordering: the CALLER makes every rank's stage A (B) of batch n complete
 * and visible before any rank's stage B (C) of that batch reads its buffer (a cross-rank barrier
 * on the stream), and keeps a receive buffer unwritten by batch n + 3 until its reader is done.
 * tdma_slab_set_peers(slab, slot, recv_of_rank, yrecv_of_rank): HOST arrays of nranks DEVICE
 * pointers, rank q's recv and yrecv buffer of ring slot `slot` (0..2; batch n uses slot n % 3);
 * copied to the device synchronously -- call it once per slot before the first batch.
 * _stage_a_peer / _stage_b_peer (pdd != 0: the PDD reduced solve) = _stage_a / _stage_b with the
 * output redirected; TDMA_ERR_INVALID_ARG before set_peers for the batch's slot. */
int tdma_slab_set_peers(tdma_slab *slab, int slot, const void *const *recv_of_rank, const void *const *yrecv_of_rank);
int tdma_slab_stage_a_peer(tdma_slab *slab, int batch_index, const void *a, const void *b, const void *c,
                           const void *d, void *stream);
int tdma_slab_stage_b_peer(tdma_slab *slab, int batch_index, const void *recv, int pdd, void *stream);
int tdma_slab_destroy(tdma_slab *slab);

/* Allocation-free solve, for callers that cannot call cudaMalloc (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid it).  Solves the same nx*ny*nz systems as tdma_solve
 * (layout and meaning of a, b, c, d, x as at the top of this file; DEVICE pointers, 8-byte aligned;
 * y split into P partitions, ny % P == 0, ny / P >= 2) with the PIPELINED variant's three stage
 * kernels run in Alg. 1 order on `stream`, batch after batch.  No plan: the
 * scratch (a', c', d' of a batch and its reduced system) is a file-scope __device__ array of
 * TDMA_STATIC_SCRATCH_BYTES that every GPU loading the library holds until the process exits, and
 * the call performs no cudaMalloc / cudaFree and no allocating library call.  The z range is cut
 * into the largest batches that fit; TDMA_ERR_UNSUPPORTED (message in tdma_last_error()) when a
 * single z-slice does not:  8 * nx * (3 ny + 10 P) bytes (+ rounding) must not exceed the maximum
 * -- e.g. 1024 x 1024 slices with P = 16 fit (25.3 MiB), 2048 x 1024 do not.
 * The array is SHARED by every call and keeps the last call's contents; nothing in it needs to be
 * zero at entry (every element read is written earlier in the same call) and nothing is cleared.
 * Calls that OVERLAP on the GPU -- different streams, independent graph branches, several host
 * threads -- race on it: order them.  The first call on a device resolves the array's device
 * address (cudaGetSymbolAddress) and, with lazy module loading, loads the kernels: make it
 * outside stream capture.  Not a fast path: use a plan when allocation is possible.  Enqueue-only. */
#define TDMA_STATIC_SCRATCH_BYTES (32u << 20)
int tdma_solve_static(int nx, int ny, int nz, int P, const void *a, const void *b, const void *c,
                      const void *d, void *x, void *stream);

/* fp64 ALU probe: measures on the current device and writes to result[0..5]
 *   [0] DFMA throughput with many independent chains, TFLOP/s (1 DFMA = 2 flop)
 *   [1] the same as DFMA per SM and cycle at the nominal SM clock
 *   [2] cycles per DEPENDENT DFMA            [3] cycles per dependent Newton reciprocal + DADD
 *   [4] cycles per dependent IEEE division + DADD       [5] nominal SM clock, MHz
 * n = capacity of result (>= 6).  Synchronises; a measurement utility for bench.py's "alu" roofline
 * of the shared-coefficient form, not part of the solve path. */
int tdma_probe_fp64(double *result, int n);

int tdma_plan_destroy(tdma_plan *plan);
const char *tdma_last_error(void); /* thread-local, never NULL */
int tdma_last_status(void);        /* thread-local: the tdma_status that came with tdma_last_error()'s message
                                      (what a failed tdma_plan_create*, which returns NULL, would have returned);
                                      TDMA_OK before the first failure */
int tdma_version(void);            /* 10000*major + 100*minor + patch */

#ifdef __cplusplus
}
#endif
#endif /* TDMA_H_ */
