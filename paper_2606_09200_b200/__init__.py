"""paper_2606_09200_b200 -- thin Python binding over libra.so (the C ABI in include/ra.h).

Argument marshalling only: every step of the hot path (GEMM, allreduce / alltoall stand-ins,
overlap schedule, sweep) runs inside the library's hand-written sm_100a kernels and its C++
driver.  PyTorch is used by callers for device memory and stream handles; this module accepts
torch tensors (or raw integer device pointers) and passes ``tensor.data_ptr()`` through.

There is no CPU fallback.  If libra.so is missing it is built with nvcc; if that fails the
import raises.  This package never imports ``oracle``.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, Structure, byref, c_char_p, c_double, c_float, c_int, c_int32, c_size_t, c_uint64, c_void_p

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))

RA_OK, RA_ERR_INVALID_ARG, RA_ERR_UNSUPPORTED, RA_ERR_INFEASIBLE_KNOB, RA_ERR_CUDA, RA_ERR_ARCH = range(6)
RA_ERR_SCRATCH_LIMIT = 6
RA_GEMM_STATIC_WS_BYTES = 16 << 20      # include/ra.h: the scratch ra_gemm_static_ws carries inside libra.so
RA_COLL_ALLREDUCE, RA_COLL_ALLTOALL, RA_COLL_NONE = 0, 1, 2
RA_MODE_SERIAL, RA_MODE_OVERLAP = 0, 1
RA_MAX_RANKS = 16
RA_DTYPE_BF16, RA_DTYPE_F32 = 0, 1

# every symbol include/ra.h declares (tests/test_abi.py checks the header against this and the .so)
EXPORTS = (
    "ra_status_str", "ra_last_cuda_error", "ra_shutdown", "ra_device_info", "ra_gemm_plan_query", "ra_gemm_residency",
    "ra_gemm_workspace_bytes", "ra_gemm", "ra_gemm_ex", "ra_gemm_static_ws", "ra_allreduce_emul", "ra_allreduce_emul_ex", "ra_alltoall_emul",
    "ra_alltoall_emul_ex",
    "ra_overlap_run", "ra_overlap_run_host", "ra_overlap_suggest", "ra_overlap_autotune", "ra_overlap_sweep", "ra_set_trace",
    "ra_l2_persist", "ra_ipc_export", "ra_ipc_open", "ra_ipc_close", "ra_peer_slice", "ra_allreduce_peer", "ra_alltoall_peer",
)


class RaError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {status_str(status)} (cuda error {last_cuda_error()})")


class Occupancy(Structure):
    _fields_ = [("smem_reserve_bytes", c_int32), ("sm_budget", c_int32), ("tiles_per_cta", c_int32),
                ("allow_clamp", c_int32), ("cta_group", c_int32), ("m_blocks", c_int32), ("cluster_k", c_int32),
                ("l2_persist_bytes", c_int32), ("tile_k", c_int32), ("tile_order", c_int32)]


class IpcHandle(Structure):
    """ra_ipc_handle: plain bytes (bytes(handle) / IpcHandle.from_buffer_copy(b)) -- ship it over any transport."""
    _fields_ = [("opaque", ctypes.c_uint8 * 64), ("offset", ctypes.c_uint64), ("bytes", ctypes.c_uint64)]


class GemmPlan(Structure):
    _fields_ = [(n, c_int32) for n in ("ctas_per_sm", "grid", "stages", "tile_m", "tile_n", "tile_k", "split_k",
                                       "swap_ab", "dyn_smem_bytes", "smem_left_per_sm", "n_tiles", "clamped", "cta_group",
                                       "m_blocks", "cluster_k", "hw_ctas_per_sm", "group_x", "l2_persist_bytes")]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


class Workload(Structure):
    _fields_ = [("transA", c_int32), ("transB", c_int32), ("M", c_int32), ("N", c_int32), ("K", c_int32),
                ("alpha", c_float), ("beta", c_float),
                ("A", c_void_p), ("lda", c_int32), ("B", c_void_p), ("ldb", c_int32), ("C", c_void_p), ("ldc", c_int32),
                ("workspace", c_void_p), ("workspace_bytes", c_size_t),
                ("kind", c_int32), ("P", c_int32), ("ar_bufs", POINTER(c_void_p)), ("ar_count", c_size_t),
                ("a2a_a", c_void_p), ("a2a_b", c_void_p), ("chunk_bytes", c_size_t), ("n_iters", c_int32),
                ("ar_pristine", POINTER(c_void_p))]


class OverlapCfg(Structure):
    _fields_ = [("mode", c_int32), ("occ", Occupancy), ("coll_sm_budget", c_int32), ("coll_smem_bytes", c_int32),
                ("coll_ctas_per_sm", c_int32), ("coll_variant", c_int32), ("prio_compute", c_int32),
                ("prio_comm", c_int32), ("dependent", c_int32), ("record_kernel_times", c_int32), ("use_graph", c_int32)]


class HostIO(Structure):
    _fields_ = [("A", c_void_p), ("B", c_void_p), ("C", c_void_p), ("ar_in", POINTER(c_void_p)), ("ar_out", c_void_p),
                ("a2a_in", c_void_p), ("a2a_out", c_void_p)]


class Peaks(Structure):
    _fields_ = [("tensor_tflops", c_double), ("hbm_gbs", c_double)]


class Suggestion(Structure):
    _fields_ = [("cfg", OverlapCfg), ("gemm_bound", c_int32), ("t_gemm_ms", c_double), ("t_coll_ms", c_double),
                ("t_overlap_ms", c_double), ("t_serial_ms", c_double), ("t_roofline_ms", c_double)]


class OverlapResult(Structure):
    _fields_ = [("total_ms", c_float), ("median_ms", c_float), ("min_ms", c_float), ("gemm_ms_sum", c_float),
                ("coll_ms_sum", c_float), ("overlap_rate", c_float), ("plan", GemmPlan),
                ("kernel_times", POINTER(c_float))]


_lib = None


def lib_path() -> str:
    return _build.LIB


def _L():
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build()  # no-op when up to date; raises if nvcc fails -- there is no fallback
    lib = ctypes.CDLL(path)
    lib.ra_status_str.restype = c_char_p
    lib.ra_status_str.argtypes = [c_int]
    lib.ra_last_cuda_error.restype = c_int
    lib.ra_shutdown.restype = None
    lib.ra_device_info.argtypes = [POINTER(c_int)] * 6
    lib.ra_gemm_plan_query.argtypes = [c_int] * 5 + [POINTER(Occupancy), POINTER(GemmPlan)]
    lib.ra_gemm_residency.argtypes = [POINTER(c_int32), c_int]
    lib.ra_gemm_workspace_bytes.restype = c_size_t
    lib.ra_gemm_workspace_bytes.argtypes = [c_int] * 5 + [POINTER(Occupancy)]
    lib.ra_gemm.argtypes = [c_int, c_int, c_int, c_int, c_int, c_float, c_void_p, c_int, c_void_p, c_int, c_float,
                            c_void_p, c_int, POINTER(Occupancy), c_void_p, c_size_t, c_void_p]
    lib.ra_gemm_ex.argtypes = [c_int, c_int, c_int, c_int, c_int, c_float, c_void_p, c_int, c_void_p, c_int, c_float,
                               c_void_p, c_int, c_int, POINTER(Occupancy), c_void_p, c_size_t, c_void_p]
    lib.ra_gemm_static_ws.argtypes = [c_int, c_int, c_int, c_int, c_int, c_float, c_void_p, c_int, c_void_p, c_int, c_float,
                                      c_void_p, c_int, POINTER(Occupancy), c_void_p]
    lib.ra_allreduce_emul.argtypes = [POINTER(c_void_p), c_int, c_size_t, c_int, c_void_p]
    lib.ra_allreduce_emul_ex.argtypes = [POINTER(c_void_p), c_int, c_size_t, c_int, c_int, c_int, c_int, c_void_p]
    lib.ra_alltoall_emul.argtypes = [c_void_p, c_void_p, c_int, c_size_t, c_int, c_void_p]
    lib.ra_alltoall_emul_ex.argtypes = [c_void_p, c_void_p, c_int, c_size_t, c_int, c_int, c_int, c_int, c_void_p]
    lib.ra_overlap_run.argtypes = [POINTER(Workload), POINTER(OverlapCfg), POINTER(OverlapResult)]
    lib.ra_overlap_run_host.argtypes = [POINTER(Workload), POINTER(Workload), POINTER(HostIO), POINTER(OverlapCfg), c_int,
                                        POINTER(OverlapResult)]
    lib.ra_overlap_suggest.argtypes = [POINTER(Workload), POINTER(Peaks), POINTER(Suggestion)]
    lib.ra_overlap_autotune.argtypes = [POINTER(Workload), POINTER(Peaks), c_int, POINTER(OverlapCfg), POINTER(OverlapResult),
                                        POINTER(c_int)]
    lib.ra_overlap_sweep.argtypes = [POINTER(Workload), POINTER(OverlapCfg), c_int, c_int, POINTER(OverlapResult),
                                     POINTER(c_int)]
    lib.ra_set_trace.argtypes = [c_void_p, c_size_t]
    lib.ra_l2_persist.argtypes = [ctypes.c_int64, POINTER(ctypes.c_int64)]
    lib.ra_ipc_export.argtypes = [c_void_p, POINTER(IpcHandle)]
    lib.ra_ipc_open.argtypes = [POINTER(IpcHandle), POINTER(c_void_p)]
    lib.ra_ipc_close.argtypes = [c_void_p]
    lib.ra_peer_slice.argtypes = [c_size_t, c_int, c_int, POINTER(c_size_t), POINTER(c_size_t)]
    lib.ra_allreduce_peer.argtypes = [POINTER(c_void_p), c_int, c_int, c_size_t, c_int, c_int, c_void_p]
    lib.ra_alltoall_peer.argtypes = [c_void_p, POINTER(c_void_p), c_int, c_int, c_size_t, c_int, c_int, c_void_p]
    for name in EXPORTS:
        fn = getattr(lib, name)
        if name not in ("ra_status_str", "ra_last_cuda_error", "ra_shutdown", "ra_gemm_workspace_bytes"):
            fn.restype = c_int
    _lib = lib
    return lib


# ---- helpers -----------------------------------------------------------------------------------
def status_str(s: int) -> str:
    return _L().ra_status_str(int(s)).decode()


def last_cuda_error() -> int:
    return int(_L().ra_last_cuda_error())


def _check(s: int, where: str):
    if s != RA_OK:
        raise RaError(s, where)


def _ptr(x) -> int | None:
    """torch tensor -> device address; int/None pass through."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return int(x.data_ptr())
    return int(x.ctypes.data)          # numpy array (host buffers of ra_overlap_run_host)


def _stream(stream) -> int | None:
    if stream is None:
        try:
            import torch
            return int(torch.cuda.current_stream().cuda_stream) or None
        except Exception:
            return None
    if isinstance(stream, int):
        return stream or None
    return int(stream.cuda_stream) or None


def _occ(occ) -> Occupancy | None:
    if occ is None or isinstance(occ, Occupancy):
        return occ
    return Occupancy(int(occ.get("smem_reserve_bytes", 0)), int(occ.get("sm_budget", 0)),
                     int(occ.get("tiles_per_cta", 0)), int(occ.get("allow_clamp", 1)), int(occ.get("cta_group", 0)),
                     int(occ.get("m_blocks", 0)), int(occ.get("cluster_k", 0)), int(occ.get("l2_persist_bytes", 0)),
                     int(occ.get("tile_k", 0)), int(occ.get("tile_order", 0)))


def _occ_ref(occ):
    o = _occ(occ)
    return byref(o) if o is not None else None


# ---- the C ABI, same names -----------------------------------------------------------------------
def ra_shutdown() -> None:
    _L().ra_shutdown()


def ra_device_info() -> dict:
    vals = [c_int(0) for _ in range(6)]
    _check(_L().ra_device_info(*[byref(v) for v in vals]), "ra_device_info")
    keys = ("sm_count", "smem_per_sm", "smem_per_block_optin", "smem_reserved_per_block", "prio_least", "prio_greatest")
    return {k: v.value for k, v in zip(keys, vals)}


def ra_gemm_plan_query(transA, transB, M, N, K, occ=None) -> dict:
    plan = GemmPlan()
    _check(_L().ra_gemm_plan_query(transA, transB, M, N, K, _occ_ref(occ), byref(plan)), "ra_gemm_plan_query")
    return plan.as_dict()


def ra_gemm_residency(reset: bool = False) -> int:
    """Largest number of GEMM CTAs seen resident on one SM at the same time since the last reset (synchronises)."""
    v = c_int32(0)
    _check(_L().ra_gemm_residency(byref(v), 1 if reset else 0), "ra_gemm_residency")
    return v.value


def ra_gemm_workspace_bytes(transA, transB, M, N, K, occ=None) -> int:
    return int(_L().ra_gemm_workspace_bytes(transA, transB, M, N, K, _occ_ref(occ)))


def ra_gemm(transA, transB, M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, occ=None, workspace=None,
            workspace_bytes=None, stream=None) -> None:
    if workspace is not None and workspace_bytes is None:
        workspace_bytes = workspace.numel() * workspace.element_size()
    _check(_L().ra_gemm(transA, transB, M, N, K, float(alpha), _ptr(A), lda, _ptr(B), ldb, float(beta), _ptr(C), ldc,
                        _occ_ref(occ), _ptr(workspace), int(workspace_bytes or 0), _stream(stream)), "ra_gemm")


def ra_gemm_ex(transA, transB, M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, c_dtype=RA_DTYPE_BF16, occ=None, workspace=None,
               workspace_bytes=None, stream=None) -> None:
    if workspace is not None and workspace_bytes is None:
        workspace_bytes = workspace.numel() * workspace.element_size()
    _check(_L().ra_gemm_ex(transA, transB, M, N, K, float(alpha), _ptr(A), lda, _ptr(B), ldb, float(beta), _ptr(C), ldc,
                           int(c_dtype), _occ_ref(occ), _ptr(workspace), int(workspace_bytes or 0), _stream(stream)), "ra_gemm_ex")


def ra_gemm_static_ws(transA, transB, M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, occ=None, stream=None) -> None:
    """ra_gemm for callers that cannot allocate device memory (a plug-in inside a host application whose pool owns the HBM,
    a serving path where cudaMalloc would stall the overlapped streams): the stream-K scratch is a fixed
    RA_GEMM_STATIC_WS_BYTES array inside libra.so.  Raises RaError(RA_ERR_SCRATCH_LIMIT) when the plan needs more.  Every
    call shares that array: do not let two of them run on the GPU at the same time.  See include/ra.h."""
    _check(_L().ra_gemm_static_ws(transA, transB, M, N, K, float(alpha), _ptr(A), lda, _ptr(B), ldb, float(beta), _ptr(C),
                                  ldc, _occ_ref(occ), _stream(stream)), "ra_gemm_static_ws")


def _ptr_array(bufs):
    arr = (c_void_p * len(bufs))(*[_ptr(b) for b in bufs])
    return arr


def ra_allreduce_emul(bufs, count=None, sm_budget=0, stream=None) -> None:
    if count is None:
        count = bufs[0].numel()
    arr = _ptr_array(bufs)
    _check(_L().ra_allreduce_emul(arr, len(bufs), int(count), int(sm_budget), _stream(stream)), "ra_allreduce_emul")


def ra_allreduce_emul_ex(bufs, count=None, sm_budget=0, ctas_per_sm=0, smem_bytes_per_cta=0, variant=0, stream=None) -> None:
    if count is None:
        count = bufs[0].numel()
    arr = _ptr_array(bufs)
    _check(_L().ra_allreduce_emul_ex(arr, len(bufs), int(count), int(sm_budget), int(smem_bytes_per_cta), int(ctas_per_sm),
                                     int(variant), _stream(stream)), "ra_allreduce_emul_ex")


def ra_alltoall_emul(send, recv, P, chunk_bytes, sm_budget=0, stream=None) -> None:
    _check(_L().ra_alltoall_emul(_ptr(send), _ptr(recv), int(P), int(chunk_bytes), int(sm_budget), _stream(stream)),
           "ra_alltoall_emul")


def ra_alltoall_emul_ex(send, recv, P, chunk_bytes, sm_budget=0, smem_bytes_per_cta=0, ctas_per_sm=0, variant=0,
                        stream=None) -> None:
    _check(_L().ra_alltoall_emul_ex(_ptr(send), _ptr(recv), int(P), int(chunk_bytes), int(sm_budget),
                                    int(smem_bytes_per_cta), int(ctas_per_sm), int(variant), _stream(stream)),
           "ra_alltoall_emul_ex")


# ---- N4: peer-memory collectives (one process per GPU; see paper_2606_09200_b200/peer.py for the handle exchange) ----
def ra_ipc_export(dev) -> bytes:
    """Handle bytes for a device tensor / pointer of this process."""
    h = IpcHandle()
    _check(_L().ra_ipc_export(_ptr(dev), byref(h)), "ra_ipc_export")
    return bytes(h)


def ra_ipc_open(handle: bytes) -> int:
    """Maps a peer's handle; returns the device pointer (int)."""
    h = IpcHandle.from_buffer_copy(handle)
    p = c_void_p(0)
    _check(_L().ra_ipc_open(byref(h), byref(p)), "ra_ipc_open")
    return int(p.value)


def ra_ipc_close(ptr: int) -> None:
    _check(_L().ra_ipc_close(c_void_p(int(ptr))), "ra_ipc_close")


def ra_peer_slice(count: int, P: int, rank: int) -> tuple:
    b, e = c_size_t(0), c_size_t(0)
    _check(_L().ra_peer_slice(int(count), int(P), int(rank), byref(b), byref(e)), "ra_peer_slice")
    return int(b.value), int(e.value)


def ra_allreduce_peer(bufs, rank, count, sm_budget=0, variant=0, stream=None) -> None:
    """bufs: the P device pointers (tensors or ints) in rank order."""
    arr = _ptr_array(bufs)
    _check(_L().ra_allreduce_peer(arr, len(bufs), int(rank), int(count), int(sm_budget), int(variant), _stream(stream)),
           "ra_allreduce_peer")


def ra_alltoall_peer(send, recv, rank, chunk_bytes, sm_budget=0, variant=0, stream=None) -> None:
    """send: this rank's P chunks; recv: the P ranks' receive buffers (tensors or ints) in rank order."""
    arr = _ptr_array(recv)
    _check(_L().ra_alltoall_peer(_ptr(send), arr, len(recv), int(rank), int(chunk_bytes), int(sm_budget), int(variant),
                                 _stream(stream)), "ra_alltoall_peer")


def ra_set_trace(buf, capacity: int = 0) -> None:
    _check(_L().ra_set_trace(_ptr(buf), int(capacity)), "ra_set_trace")


def make_workload(*, gemm=None, allreduce=None, alltoall=None, n_iters=1, ar_pristine=None):
    """Marshal a workload.  gemm = dict(M,N,K,A,B,C[,alpha,beta,lda,ldb,ldc,transA,transB,workspace]);
    allreduce = list of P fp32 tensors; alltoall = dict(a, b, P, chunk_bytes); ar_pristine = optional list of P
    fp32 tensors the library copies into the allreduce buffers before every run (outside the timed window).
    Returns (Workload, keepalive) -- keepalive holds the pointer array."""
    w = Workload()
    keep = []
    if gemm is not None:
        g = gemm
        w.transA, w.transB = int(g.get("transA", 0)), int(g.get("transB", 1))
        w.M, w.N, w.K = int(g["M"]), int(g["N"]), int(g["K"])
        w.alpha, w.beta = float(g.get("alpha", 1.0)), float(g.get("beta", 0.0))
        w.A, w.B, w.C = _ptr(g["A"]), _ptr(g["B"]), _ptr(g["C"])
        w.lda = int(g.get("lda", w.M if w.transA else w.K))
        w.ldb = int(g.get("ldb", w.K if w.transB else w.N))
        w.ldc = int(g.get("ldc", w.N))
        ws = g.get("workspace")
        if ws is not None:
            w.workspace = _ptr(ws)
            w.workspace_bytes = ws.numel() * ws.element_size()
    if allreduce is not None:
        arr = _ptr_array(allreduce)
        keep.append(arr)
        w.kind, w.P = RA_COLL_ALLREDUCE, len(allreduce)
        w.ar_bufs = ctypes.cast(arr, POINTER(c_void_p))
        w.ar_count = int(allreduce[0].numel())
        if ar_pristine is not None:
            assert len(ar_pristine) == len(allreduce)
            parr = _ptr_array(ar_pristine)
            keep.append(parr)
            w.ar_pristine = ctypes.cast(parr, POINTER(c_void_p))
    elif alltoall is not None:
        w.kind, w.P = RA_COLL_ALLTOALL, int(alltoall["P"])
        w.a2a_a, w.a2a_b = _ptr(alltoall["a"]), _ptr(alltoall["b"])
        w.chunk_bytes = int(alltoall["chunk_bytes"])
    else:
        w.kind = RA_COLL_NONE
    w.n_iters = int(n_iters)
    return w, keep


def make_cfg(mode=RA_MODE_OVERLAP, occ=None, coll_sm_budget=0, coll_smem_bytes=0, coll_ctas_per_sm=0, coll_variant=0,
             prio_compute=0, prio_comm=0, dependent=1, record_kernel_times=0, use_graph=0) -> OverlapCfg:
    c = OverlapCfg()
    c.mode = int(mode)
    c.occ = _occ(occ) or Occupancy(0, 0, 0, 1, 0)
    c.coll_sm_budget, c.coll_smem_bytes = int(coll_sm_budget), int(coll_smem_bytes)
    c.coll_ctas_per_sm, c.coll_variant = int(coll_ctas_per_sm), int(coll_variant)
    c.prio_compute, c.prio_comm = int(prio_compute), int(prio_comm)
    c.dependent, c.record_kernel_times = int(dependent), int(record_kernel_times)
    c.use_graph = int(use_graph)
    return c


def _result_dict(r: OverlapResult, n_iters: int, times) -> dict:
    d = {"total_ms": r.total_ms, "median_ms": r.median_ms, "min_ms": r.min_ms, "gemm_ms_sum": r.gemm_ms_sum,
         "coll_ms_sum": r.coll_ms_sum, "overlap_rate": r.overlap_rate, "plan": r.plan.as_dict()}
    if times is not None:
        d["kernel_times"] = [list(times[4 * i:4 * i + 4]) for i in range(n_iters)]
    return d


def ra_overlap_run(workload: Workload, cfg: OverlapCfg) -> dict:
    res = OverlapResult()
    times = None
    if cfg.record_kernel_times:
        times = (c_float * (4 * workload.n_iters))()
        res.kernel_times = ctypes.cast(times, POINTER(c_float))
    _check(_L().ra_overlap_run(byref(workload), byref(cfg), byref(res)), "ra_overlap_run")
    return _result_dict(res, workload.n_iters, times)


def make_host_io(*, A=None, B=None, C=None, ar_in=None, ar_out=None, a2a_in=None, a2a_out=None):
    """Marshal the HOST buffers of one step (pinned torch CPU tensors or numpy arrays).  Returns (HostIO, keepalive)."""
    io = HostIO()
    keep = [A, B, C, ar_in, ar_out, a2a_in, a2a_out]
    io.A, io.B, io.C = _ptr(A), _ptr(B), _ptr(C)
    if ar_in is not None:
        arr = _ptr_array(ar_in)
        keep.append(arr)
        io.ar_in = ctypes.cast(arr, POINTER(c_void_p))
    io.ar_out, io.a2a_in, io.a2a_out = _ptr(ar_out), _ptr(a2a_in), _ptr(a2a_out)
    return io, keep


def ra_l2_persist(nbytes: int) -> int:
    """Sets the device's persisting-L2 carve-out (0 = give it back); returns the bytes granted."""
    from ctypes import c_int64
    g = c_int64(0)
    _check(_L().ra_l2_persist(c_int64(int(nbytes)), byref(g)), "ra_l2_persist")
    return int(g.value)


def ra_overlap_run_host(dev0: Workload, dev1, io: HostIO, cfg: OverlapCfg, n_steps: int = 1) -> dict:
    """n_steps steps from host buffers, copies pipelined against compute over the device sets dev0 / dev1 (or None)."""
    res = OverlapResult()
    _check(_L().ra_overlap_run_host(byref(dev0), byref(dev1) if dev1 is not None else None, byref(io), byref(cfg),
                                    int(n_steps), byref(res)), "ra_overlap_run_host")
    return _result_dict(res, dev0.n_iters, None)


def cfg_to_kw(c: OverlapCfg) -> dict:
    """OverlapCfg -> the keyword form make_cfg takes (for logging / re-creating a setting)."""
    return dict(mode=c.mode, occ=dict(smem_reserve_bytes=c.occ.smem_reserve_bytes, sm_budget=c.occ.sm_budget,
                                      tiles_per_cta=c.occ.tiles_per_cta, cta_group=c.occ.cta_group, m_blocks=c.occ.m_blocks,
                                      cluster_k=c.occ.cluster_k, l2_persist_bytes=c.occ.l2_persist_bytes, tile_k=c.occ.tile_k, tile_order=c.occ.tile_order),
                coll_sm_budget=c.coll_sm_budget, coll_smem_bytes=c.coll_smem_bytes, coll_ctas_per_sm=c.coll_ctas_per_sm,
                coll_variant=c.coll_variant, prio_compute=c.prio_compute, prio_comm=c.prio_comm, dependent=c.dependent,
                use_graph=c.use_graph)


def ra_overlap_suggest(workload: Workload, tensor_tflops: float = 0.0, hbm_gbs: float = 0.0) -> dict:
    """Model-based knob policy (host only).  Returns {"cfg": OverlapCfg, "kw": make_cfg keywords, predictions...}."""
    s = Suggestion()
    pk = Peaks(float(tensor_tflops), float(hbm_gbs))
    _check(_L().ra_overlap_suggest(byref(workload), byref(pk), byref(s)), "ra_overlap_suggest")
    kw = cfg_to_kw(s.cfg)
    return {"kw": kw, "gemm_bound": "hbm" if s.gemm_bound else "tensor", "t_gemm_ms": s.t_gemm_ms, "t_coll_ms": s.t_coll_ms,
            "t_overlap_ms": s.t_overlap_ms, "t_serial_ms": s.t_serial_ms, "t_roofline_ms": s.t_roofline_ms}


def ra_overlap_autotune(workload: Workload, tensor_tflops: float = 0.0, hbm_gbs: float = 0.0, runs: int = 9):
    """Model pick + neighbours, measured.  Returns (best OverlapCfg, its result dict, number of settings timed)."""
    pk = Peaks(float(tensor_tflops), float(hbm_gbs))
    cfg, res, n = OverlapCfg(), OverlapResult(), c_int(0)
    _check(_L().ra_overlap_autotune(byref(workload), byref(pk), int(runs), byref(cfg), byref(res), byref(n)),
           "ra_overlap_autotune")
    return cfg, _result_dict(res, workload.n_iters, None), n.value


def ra_overlap_sweep(workload: Workload, cfgs, runs: int = 30):
    """Returns (list of result dicts, best index)."""
    n = len(cfgs)
    carr = (OverlapCfg * n)(*cfgs)
    rarr = (OverlapResult * n)()
    keep = []
    for i in range(n):
        if cfgs[i].record_kernel_times:
            t = (c_float * (4 * workload.n_iters))()
            keep.append(t)
            rarr[i].kernel_times = ctypes.cast(t, POINTER(c_float))
        else:
            keep.append(None)
    best = c_int(-1)
    _check(_L().ra_overlap_sweep(byref(workload), carr, n, int(runs), rarr, byref(best)), "ra_overlap_sweep")
    return [_result_dict(rarr[i], workload.n_iters, keep[i]) for i in range(n)], best.value
