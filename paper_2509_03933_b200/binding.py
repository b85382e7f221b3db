"""Thin Python binding of the C ABI in ``include/tdma.h`` (argument marshalling only).

Same names as the C entry points: ``tdma_plan_create``, ``tdma_plan_create_ex``, ``tdma_solve``,
``tdma_solve_host``, ``tdma_stage``, ``tdma_plan_get``, ``tdma_plan_workspace_bytes``,
``tdma_plan_buffer``, ``tdma_plan_destroy``, ``tdma_last_error``, ``tdma_version``, ``tdma_solve_shared``,
``tdma_slab_*``, ``tdma_probe_fp64``, ... (``EXPORTED_SYMBOLS``) -- plus a small ``Plan`` convenience class.  Every step of the path runs inside ``libtdma.so``'s kernels; PyTorch
is used by callers only for device memory and streams.  There is no CPU fallback: if the shared
library is missing (and cannot be built) importing a compute entry point raises.
"""
from __future__ import annotations

import ctypes
import os
import sys
from typing import Optional

from . import build as _build

# enums of include/tdma.h
TDMA_F64 = 0
TDMA_OK, TDMA_ERR_INVALID_ARG, TDMA_ERR_UNSUPPORTED, TDMA_ERR_ALLOC, TDMA_ERR_CUDA = 0, -1, -2, -3, -4
TDMA_VARIANT_AUTO, TDMA_VARIANT_PIPELINED, TDMA_VARIANT_FUSED, TDMA_VARIANT_STAGED = 0, 1, 2, 3
TDMA_AXIS_Y, TDMA_AXIS_X, TDMA_AXIS_Z = 0, 1, 2
TDMA_STAGE_A, TDMA_STAGE_GATHER, TDMA_STAGE_B, TDMA_STAGE_C = 0, 1, 2, 3
(TDMA_GET_NB, TDMA_GET_M, TDMA_GET_BATCH, TDMA_GET_NSTREAMS, TDMA_GET_DEPTH, TDMA_GET_VARIANT,
 TDMA_GET_LAUNCHES, TDMA_GET_FUSED_LINES, TDMA_GET_FUSED_CLUSTER, TDMA_GET_GRAPH_BUILDS,
 TDMA_GET_FUSED_LEAF_ROWS, TDMA_GET_FUSED_TOP, TDMA_GET_FUSED_THREADS, TDMA_GET_FUSED_SMEM,
 TDMA_GET_FUSED_TOP_ROWS, TDMA_GET_FUSED_IMPL, TDMA_GET_FUSED_FILL, TDMA_GET_SHARED_LINES,
 TDMA_GET_SHARED_CLUSTER, TDMA_GET_SHARED_LEAF_ROWS, TDMA_GET_SHARED_THREADS, TDMA_GET_SHARED_SMEM,
 TDMA_GET_SHARED_SLOTS, TDMA_GET_SHARED_FILL, TDMA_GET_REDUCED_PARTITIONS, TDMA_GET_SHARED_LINE_KERNEL) = range(26)
(TDMA_BUF_RA, TDMA_BUF_RC, TDMA_BUF_RD, TDMA_BUF_Y, TDMA_BUF_SA, TDMA_BUF_SC, TDMA_BUF_SD) = range(7)

EXPORTED_SYMBOLS = (
    "tdma_plan_create", "tdma_plan_create_ex", "tdma_solve", "tdma_solve_host", "tdma_stage",
    "tdma_plan_get", "tdma_plan_workspace_bytes", "tdma_plan_buffer", "tdma_plan_destroy",
    "tdma_last_error", "tdma_last_status", "tdma_version", "tdma_pipeline_model", "tdma_plan_autotune", "tdma_plan_timeline",
    "tdma_solve_shared", "tdma_probe_fp64", "tdma_solve_static",
    "tdma_slab_create", "tdma_slab_get", "tdma_slab_stage_a", "tdma_slab_stage_b", "tdma_slab_stage_b_pdd", "tdma_slab_stage_c",
    "tdma_slab_set_peers", "tdma_slab_stage_a_peer", "tdma_slab_stage_b_peer", "tdma_slab_destroy",
)
(TDMA_SLAB_NB, TDMA_SLAB_BATCH, TDMA_SLAB_LINES, TDMA_SLAB_SHARE, TDMA_SLAB_PTOT, TDMA_SLAB_PLOCAL,
 TDMA_SLAB_TMA) = range(7)


class tdma_options(ctypes.Structure):
    _fields_ = [
        ("struct_size", ctypes.c_int), ("variant", ctypes.c_int), ("nstreams", ctypes.c_int),
        ("use_graph", ctypes.c_int), ("separate_gather", ctypes.c_int),
        ("fused_lines", ctypes.c_int), ("fused_cluster", ctypes.c_int),
        ("fused_leaf_rows", ctypes.c_int), ("fused_top", ctypes.c_int),
        ("fused_impl", ctypes.c_int), ("fused_fill", ctypes.c_int), ("axis", ctypes.c_int), ("periodic", ctypes.c_int),
        ("timeline", ctypes.c_int), ("fused_slots", ctypes.c_int), ("host_chunk", ctypes.c_int),
        ("shared_lines", ctypes.c_int), ("shared_cluster", ctypes.c_int), ("shared_leaf_rows", ctypes.c_int),
        ("shared_slots", ctypes.c_int), ("pdd", ctypes.c_int), ("shared_ctas", ctypes.c_int),
    ]


class TdmaError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__("tdma error %d: %s" % (status, message))
        self.status = status


_lib: Optional[ctypes.CDLL] = None


def library_path() -> str:
    return _build.LIB_PATH


def load_library(build_if_missing: bool = True) -> ctypes.CDLL:
    """dlopen libtdma.so (building it with nvcc first if it is missing or stale)."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB_PATH
    if build_if_missing:
        try:
            path = _build.build()
        except Exception as exc:
            if not os.path.exists(path):
                raise RuntimeError("libtdma.so is missing and could not be built: %s" % exc)
            # never silent: the library on disk is older than the sources
            sys.stderr.write("paper_2509_03933_b200: WARNING: rebuilding libtdma.so failed (%s); "
                             "loading the STALE library at %s\n" % (str(exc).splitlines()[0], path))
    if not os.path.exists(path):
        raise RuntimeError("libtdma.so not found at %s (run __graft_entry__.build())" % path)
    lib = ctypes.CDLL(path)
    vp, ci, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_size_t
    lib.tdma_plan_create.argtypes = [ci] * 6
    lib.tdma_plan_create.restype = vp
    lib.tdma_plan_create_ex.argtypes = [ci] * 6 + [ctypes.POINTER(tdma_options)]
    lib.tdma_plan_create_ex.restype = vp
    lib.tdma_solve.argtypes = [vp] * 7
    lib.tdma_solve.restype = ci
    lib.tdma_solve_shared.argtypes = [vp] * 6 + [ci, ci] + [vp] * 3
    lib.tdma_solve_shared.restype = ci
    lib.tdma_slab_create.argtypes = [ci] * 7
    lib.tdma_slab_create.restype = vp
    lib.tdma_slab_get.argtypes = [vp, ci]
    lib.tdma_slab_get.restype = ci
    lib.tdma_slab_stage_a.argtypes = [vp, ci] + [vp] * 6
    lib.tdma_slab_stage_a.restype = ci
    lib.tdma_slab_stage_b.argtypes = [vp, ci] + [vp] * 3
    lib.tdma_slab_stage_b.restype = ci
    lib.tdma_slab_stage_b_pdd.argtypes = [vp, ci] + [vp] * 3
    lib.tdma_slab_stage_b_pdd.restype = ci
    lib.tdma_slab_stage_c.argtypes = [vp, ci] + [vp] * 3
    lib.tdma_slab_stage_c.restype = ci
    lib.tdma_slab_set_peers.argtypes = [vp, ci, ctypes.POINTER(vp), ctypes.POINTER(vp)]
    lib.tdma_slab_set_peers.restype = ci
    lib.tdma_slab_stage_a_peer.argtypes = [vp, ci] + [vp] * 5
    lib.tdma_slab_stage_a_peer.restype = ci
    lib.tdma_slab_stage_b_peer.argtypes = [vp, ci, vp, ci, vp]
    lib.tdma_slab_stage_b_peer.restype = ci
    lib.tdma_slab_destroy.argtypes = [vp]
    lib.tdma_slab_destroy.restype = ci
    lib.tdma_solve_static.argtypes = [ci] * 4 + [vp] * 6
    lib.tdma_solve_static.restype = ci
    lib.tdma_probe_fp64.argtypes = [ctypes.POINTER(ctypes.c_double), ci]
    lib.tdma_probe_fp64.restype = ci
    lib.tdma_solve_host.argtypes = [vp] * 6
    lib.tdma_solve_host.restype = ci
    lib.tdma_stage.argtypes = [vp, ci, ci] + [vp] * 6
    lib.tdma_stage.restype = ci
    lib.tdma_plan_get.argtypes = [vp, ci]
    lib.tdma_plan_get.restype = ci
    lib.tdma_plan_workspace_bytes.argtypes = [vp]
    lib.tdma_plan_workspace_bytes.restype = sz
    lib.tdma_plan_buffer.argtypes = [vp, ci, ci, ctypes.POINTER(vp), ctypes.POINTER(sz)]
    lib.tdma_plan_buffer.restype = ci
    lib.tdma_plan_destroy.argtypes = [vp]
    lib.tdma_plan_destroy.restype = ci
    lib.tdma_last_error.argtypes = []
    lib.tdma_last_error.restype = ctypes.c_char_p
    lib.tdma_last_status.argtypes = []
    lib.tdma_last_status.restype = ctypes.c_int
    lib.tdma_version.argtypes = []
    lib.tdma_version.restype = ci
    lib.tdma_plan_timeline.argtypes = [vp, ctypes.POINTER(ctypes.c_double), ci]
    lib.tdma_plan_timeline.restype = ci
    lib.tdma_pipeline_model.argtypes = [ci, ctypes.c_double, ctypes.c_double, ctypes.c_double, ci, ctypes.c_double]
    lib.tdma_pipeline_model.restype = ctypes.c_double
    lib.tdma_plan_autotune.argtypes = [ci] * 6 + [ctypes.POINTER(ci), ci] + [vp] * 5 + [
        ctypes.POINTER(ci), ctypes.POINTER(ctypes.c_double)]
    lib.tdma_plan_autotune.restype = ci
    _lib = lib
    return lib


def tdma_last_error() -> str:
    return load_library().tdma_last_error().decode("utf-8", "replace")


def tdma_last_status() -> int:
    return int(load_library().tdma_last_status())


def tdma_version() -> int:
    return int(load_library().tdma_version())


def _check(status: int) -> int:
    if status != TDMA_OK:
        raise TdmaError(status, tdma_last_error())
    return status


def _ptr(t) -> int:
    """Device (or host) address of a torch tensor / numpy array / int."""
    if isinstance(t, int):
        return t
    if hasattr(t, "data_ptr"):
        return int(t.data_ptr())
    if hasattr(t, "ctypes"):
        return int(t.ctypes.data)
    raise TypeError("cannot take the address of %r" % type(t))


def _stream_handle(stream) -> int:
    if stream is None:
        import torch
        return int(torch.cuda.current_stream().cuda_stream)
    if isinstance(stream, int):
        return stream
    return int(stream.cuda_stream)


def tdma_plan_create(nx: int, ny: int, nz: int, P: int, batch: int, dtype: int = TDMA_F64) -> int:
    h = load_library().tdma_plan_create(nx, ny, nz, P, batch, dtype)
    if not h:
        raise TdmaError(tdma_last_status() or TDMA_ERR_INVALID_ARG, tdma_last_error())
    return int(h)


def tdma_plan_create_ex(nx: int, ny: int, nz: int, P: int, batch: int, dtype: int = TDMA_F64, *,
                        variant: int = 0, nstreams: int = 0, use_graph: int = 0,
                        separate_gather: int = 0, fused_lines: int = 0, fused_cluster: int = 0,
                        fused_leaf_rows: int = 0, fused_top: int = 0, fused_impl: int = 0, fused_fill: int = 0,
                        axis: int = 0, periodic: int = 0, timeline: int = 0, fused_slots: int = 0, host_chunk: int = 0,
                        shared_lines: int = 0, shared_cluster: int = 0, shared_leaf_rows: int = 0,
                        shared_slots: int = 0, shared_ctas: int = 0, pdd: int = 0) -> int:
    opt = tdma_options()
    opt.struct_size = ctypes.sizeof(tdma_options)
    opt.variant, opt.nstreams, opt.use_graph = variant, nstreams, use_graph
    opt.separate_gather, opt.fused_lines, opt.fused_cluster = separate_gather, fused_lines, fused_cluster
    opt.fused_leaf_rows, opt.fused_top, opt.fused_impl = fused_leaf_rows, fused_top, fused_impl
    opt.fused_fill, opt.axis, opt.periodic, opt.timeline = fused_fill, axis, periodic, timeline
    opt.host_chunk, opt.fused_slots = host_chunk, fused_slots
    opt.shared_lines, opt.shared_cluster, opt.shared_leaf_rows, opt.shared_slots = shared_lines, shared_cluster, shared_leaf_rows, shared_slots
    opt.shared_ctas, opt.pdd = shared_ctas, pdd
    h = load_library().tdma_plan_create_ex(nx, ny, nz, P, batch, dtype, ctypes.byref(opt))
    if not h:
        raise TdmaError(tdma_last_status() or TDMA_ERR_INVALID_ARG, tdma_last_error())
    return int(h)


def tdma_solve(plan: int, a, b, c, d, x, stream=None) -> None:
    _check(load_library().tdma_solve(plan, _ptr(a), _ptr(b), _ptr(c), _ptr(d), _ptr(x),
                                     _stream_handle(stream)))


def tdma_solve_shared(plan: int, a_y, b0_y, c_y, sx, sz, ncomp: int, pin00: int, d, x, stream=None) -> None:
    _check(load_library().tdma_solve_shared(plan, _ptr(a_y), _ptr(b0_y), _ptr(c_y), _ptr(sx), _ptr(sz),
                                            int(ncomp), int(pin00), _ptr(d), _ptr(x), _stream_handle(stream)))


def tdma_slab_create(nx: int, ny_local: int, nz: int, P_local: int, batch: int, rank: int, nranks: int) -> int:
    h = load_library().tdma_slab_create(nx, ny_local, nz, P_local, batch, rank, nranks)
    if not h:
        raise TdmaError(TDMA_ERR_INVALID_ARG, "tdma_slab_create failed (invalid shape for %d ranks, no CUDA device, "
                                              "or out of memory)" % nranks)
    return int(h)


def tdma_slab_get(slab: int, what: int) -> int:
    v = int(load_library().tdma_slab_get(slab, what))
    if v < 0:
        raise TdmaError(v, "tdma_slab_get(%d)" % what)
    return v


def tdma_slab_stage_a(slab: int, batch_index: int, a, b, c, d, send, stream=None) -> None:
    _check(load_library().tdma_slab_stage_a(slab, batch_index, _ptr(a), _ptr(b), _ptr(c), _ptr(d), _ptr(send),
                                            _stream_handle(stream)))


def tdma_slab_stage_b(slab: int, batch_index: int, recv, yout, stream=None) -> None:
    _check(load_library().tdma_slab_stage_b(slab, batch_index, _ptr(recv), _ptr(yout), _stream_handle(stream)))


def tdma_slab_stage_b_pdd(slab: int, batch_index: int, recv, yout, stream=None) -> None:
    _check(load_library().tdma_slab_stage_b_pdd(slab, batch_index, _ptr(recv), _ptr(yout), _stream_handle(stream)))


def tdma_slab_stage_c(slab: int, batch_index: int, yrecv, x, stream=None) -> None:
    _check(load_library().tdma_slab_stage_c(slab, batch_index, _ptr(yrecv), _ptr(x), _stream_handle(stream)))


def tdma_slab_set_peers(slab: int, slot: int, recv_of_rank, yrecv_of_rank) -> None:
    """recv_of_rank / yrecv_of_rank: per rank, a tensor or an integer device address."""
    addr = lambda t: int(t) if isinstance(t, int) else int(t.data_ptr())
    n = len(recv_of_rank)
    if len(yrecv_of_rank) != n:
        raise ValueError("one recv and one yrecv buffer per rank")
    r = (ctypes.c_void_p * n)(*[addr(t) for t in recv_of_rank])
    y = (ctypes.c_void_p * n)(*[addr(t) for t in yrecv_of_rank])
    _check(load_library().tdma_slab_set_peers(slab, slot, r, y))


def tdma_slab_stage_a_peer(slab: int, batch_index: int, a, b, c, d, stream=None) -> None:
    _check(load_library().tdma_slab_stage_a_peer(slab, batch_index, _ptr(a), _ptr(b), _ptr(c), _ptr(d),
                                                 _stream_handle(stream)))


def tdma_slab_stage_b_peer(slab: int, batch_index: int, recv, pdd: bool = False, stream=None) -> None:
    _check(load_library().tdma_slab_stage_b_peer(slab, batch_index, _ptr(recv), 1 if pdd else 0, _stream_handle(stream)))


def tdma_slab_destroy(slab: int) -> None:
    _check(load_library().tdma_slab_destroy(slab))


TDMA_STATIC_SCRATCH_BYTES = 32 << 20


def tdma_solve_static(nx: int, ny: int, nz: int, P: int, a, b, c, d, x, stream=None) -> None:
    """Allocation-free solve (include/tdma.h): scratch in a static device array of TDMA_STATIC_SCRATCH_BYTES."""
    _check(load_library().tdma_solve_static(nx, ny, nz, P, _ptr(a), _ptr(b), _ptr(c), _ptr(d), _ptr(x),
                                            _stream_handle(stream)))


def tdma_probe_fp64() -> dict:
    """fp64 ALU probe of the current device (include/tdma.h)."""
    r = (ctypes.c_double * 6)()
    _check(load_library().tdma_probe_fp64(r, 6))
    keys = ("dfma_tflops", "dfma_per_sm_cycle", "dfma_latency_cycles", "rcp_nr_latency_cycles",
            "div_latency_cycles", "sm_clock_mhz")
    return dict(zip(keys, [float(v) for v in r]))


def tdma_solve_host(plan: int, a, b, c, d, x) -> None:
    _check(load_library().tdma_solve_host(plan, _ptr(a), _ptr(b), _ptr(c), _ptr(d), _ptr(x)))


def tdma_stage(plan: int, stage: int, batch_index: int, a, b, c, d, x, stream=None) -> None:
    _check(load_library().tdma_stage(plan, stage, batch_index, _ptr(a), _ptr(b), _ptr(c), _ptr(d),
                                     _ptr(x), _stream_handle(stream)))


def tdma_plan_get(plan: int, what: int) -> int:
    v = int(load_library().tdma_plan_get(plan, what))
    if v < 0:
        raise TdmaError(v, tdma_last_error())
    return v


def tdma_plan_workspace_bytes(plan: int) -> int:
    return int(load_library().tdma_plan_workspace_bytes(plan))


def tdma_plan_buffer(plan: int, which: int, slot: int = 0):
    """(device address, bytes) of a plan-owned stage buffer."""
    p, n = ctypes.c_void_p(), ctypes.c_size_t()
    _check(load_library().tdma_plan_buffer(plan, which, slot, ctypes.byref(p), ctypes.byref(n)))
    return int(p.value), int(n.value)


def tdma_plan_timeline(plan: int, max_launches: int = 1 << 16):
    """[(stage, batch, start_ms, end_ms)] of the last solve of a plan created with timeline=1."""
    buf = (ctypes.c_double * (4 * max_launches))()
    n = int(load_library().tdma_plan_timeline(plan, buf, max_launches))
    if n < 0:
        raise TdmaError(n, tdma_last_error())
    return [(int(buf[4 * i]), int(buf[4 * i + 1]), float(buf[4 * i + 2]), float(buf[4 * i + 3])) for i in range(n)]


def tdma_pipeline_model(nb: int, tA: float, tB: float, tC: float, nstreams: int = 2,
                        last_frac: float = 1.0) -> float:
    return float(load_library().tdma_pipeline_model(nb, tA, tB, tC, nstreams, last_frac))


def tdma_plan_autotune(nx: int, ny: int, nz: int, P: int, candidates, a, b, c, d, x, nstreams: int = 2,
                       dtype: int = TDMA_F64):
    """(best batch size, [estimated ms per candidate])."""
    n = len(candidates)
    cand = (ctypes.c_int * n)(*candidates)
    est = (ctypes.c_double * n)()
    best = ctypes.c_int(0)
    _check(load_library().tdma_plan_autotune(nx, ny, nz, P, dtype, nstreams, cand, n, _ptr(a), _ptr(b),
                                             _ptr(c), _ptr(d), _ptr(x), ctypes.byref(best), est))
    return int(best.value), [float(v) for v in est]


def tdma_plan_destroy(plan: int) -> None:
    _check(load_library().tdma_plan_destroy(plan))


class Plan:
    """RAII wrapper: ``Plan(nx, ny, nz, P, batch).solve(a, b, c, d, x)``."""

    def __init__(self, nx: int, ny: int, nz: int, P: int, batch: int = 0, **options):
        self.shape = (nz, ny, nx)
        self.P = P
        self.axis = options.get("axis", TDMA_AXIS_Y)
        self.handle = (tdma_plan_create_ex(nx, ny, nz, P, batch, TDMA_F64, **options)
                       if options else tdma_plan_create(nx, ny, nz, P, batch, TDMA_F64))

    def _validate(self, tensors):
        n = self.shape[0] * self.shape[1] * self.shape[2]
        for t in tensors:
            if hasattr(t, "numel"):
                if t.numel() != n or not t.is_contiguous() or t.element_size() != 8:
                    raise ValueError("arrays must be contiguous fp64 with nz*ny*nx elements")

    def solve(self, a, b, c, d, x, stream=None):
        self._validate((a, b, c, d, x))
        tdma_solve(self.handle, a, b, c, d, x, stream)
        return x

    def solve_shared(self, a_y, b0_y, c_y, sx, sz, d, x, pin00: bool = False, stream=None):
        """Shared-coefficient solve; d, x real (nz, ny, nx) fp64 or complex128 tensors.  sx = sz = None:
        the same matrix for every line (uniform matrix, include/tdma.h)."""
        nz, ny, nx = self.shape
        ncomp = 2 if (hasattr(d, "is_complex") and d.is_complex()) else 1
        # (line length, lines side by side, slices): z sweep: lines along z, y-slices; x sweep: lines along x,
        # ny of them per z-slice
        nline, nlane, nslice = {TDMA_AXIS_Z: (nz, nx, ny), TDMA_AXIS_X: (nx, ny, nz)}.get(self.axis, (ny, nx, nz))
        if (sx is None) != (sz is None):
            raise ValueError("pass both shift arrays, or None for both (uniform matrix)")
        for t, n in ((a_y, nline), (b0_y, nline), (c_y, nline)) + (((sx, nlane), (sz, nslice)) if sx is not None else ()):
            if t.numel() != n or not t.is_contiguous() or t.element_size() != 8:
                raise ValueError("coefficient arrays must be contiguous fp64 of lengths n, n, n (line length), lanes, slices")
        for t in (d, x):
            if t.numel() != nz * ny * nx or not t.is_contiguous() or t.element_size() != 8 * ncomp:
                raise ValueError("d, x must be contiguous with nz*ny*nx cells of %d bytes" % (8 * ncomp))
        tdma_solve_shared(self.handle, a_y, b0_y, c_y, 0 if sx is None else sx, 0 if sz is None else sz, ncomp,
                          1 if pin00 else 0, d, x, stream)
        return x

    def solve_host(self, a, b, c, d, x):
        self._validate((a, b, c, d, x))
        tdma_solve_host(self.handle, a, b, c, d, x)
        return x

    def stage(self, stage: int, batch_index: int, a, b, c, d, x, stream=None):
        tdma_stage(self.handle, stage, batch_index, a, b, c, d, x, stream)

    def timeline(self):
        return tdma_plan_timeline(self.handle)

    def get(self, what: int) -> int:
        return tdma_plan_get(self.handle, what)

    @property
    def workspace_bytes(self) -> int:
        return tdma_plan_workspace_bytes(self.handle)

    def buffer(self, which: int, slot: int = 0):
        return tdma_plan_buffer(self.handle, which, slot)

    def close(self):
        if getattr(self, "handle", None):
            h, self.handle = self.handle, None
            tdma_plan_destroy(h)

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
