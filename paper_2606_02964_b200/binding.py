"""Thin ctypes binding of libmsa.so -- same names as include/msa.h, argument marshalling only.

Every step of the hot path runs inside the library's CUDA kernels.  PyTorch appears only as
the owner of device memory and streams (``tensor.data_ptr()``, ``torch.cuda.current_stream``).
There is no fallback: if libmsa.so is missing or no sm_100 GPU is present, calls raise.
"""
from __future__ import annotations

import ctypes
import os
from typing import Dict, Optional, Tuple

import numpy as np

from ._build import LIB_PATH

MSA_OK = 0
MSA_ERR_INVALID_ARG, MSA_ERR_UNSUPPORTED, MSA_ERR_OVERLAP, MSA_ERR_UNSORTED = -1, -2, -3, -4
MSA_ERR_OUT_OF_RANGE, MSA_ERR_MISALIGNED, MSA_ERR_WORKSPACE, MSA_ERR_CUDA, MSA_ERR_NO_DEVICE = -5, -6, -7, -8, -9
MSA_ERR_STATIC_WS = -10
MSA_STATIC_WS_BYTES = 32 << 20
MSA_SEG_PAGED, MSA_SEG_CONTIG, MSA_SEG_SELF = 0, 1, 2
MSA_POOL_BF16, MSA_POOL_FP8_E4M3 = 0, 1


class MsaConfig(ctypes.Structure):
    _fields_ = [("num_q_heads", ctypes.c_int32), ("num_kv_heads", ctypes.c_int32), ("head_dim", ctypes.c_int32),
                ("block_size", ctypes.c_int32), ("q_to_kv_head", ctypes.POINTER(ctypes.c_int32)),
                ("device", ctypes.c_int32), ("pool_format", ctypes.c_int32),
                ("k_scale", ctypes.POINTER(ctypes.c_float)), ("v_scale", ctypes.POINTER(ctypes.c_float))]


class MsaSegment(ctypes.Structure):
    _fields_ = [("kind", ctypes.c_int32), ("abs_start", ctypes.c_int32), ("len", ctypes.c_int32),
                ("block_off", ctypes.c_int32), ("row_off", ctypes.c_int64)]


class MsaRequest(ctypes.Structure):
    _fields_ = [("q_row_start", ctypes.c_int32), ("q_len", ctypes.c_int32), ("q_abs_start", ctypes.c_int32),
                ("seg_begin", ctypes.c_int32), ("seg_count", ctypes.c_int32)]


class MsaPlanInfo(ctypes.Structure):
    _fields_ = [("num_ctas", ctypes.c_int32), ("num_items", ctypes.c_int32), ("num_units", ctypes.c_int32),
                ("num_split_items", ctypes.c_int32), ("num_partials", ctypes.c_int32),
                ("rows_per_tile", ctypes.c_int32), ("kv_tiles", ctypes.c_int64), ("visible_pairs", ctypes.c_int64),
                ("max_block_table_index", ctypes.c_int64), ("max_contig_row", ctypes.c_int64),
                ("max_q_row", ctypes.c_int64)]


class MsaError(RuntimeError):
    def __init__(self, status: int, where: str):
        lib = _lib()
        msg = lib.msa_strerror(status).decode()
        cuda = lib.msa_last_cuda_error().decode()
        super().__init__(f"{where}: {msg} ({status})" + (f" [{cuda}]" if cuda and status == MSA_ERR_CUDA else ""))
        self.status = status


_LIB: Optional[ctypes.CDLL] = None

EXPORTS = ["msa_create", "msa_destroy", "msa_plan_create", "msa_plan_destroy", "msa_plan_get_info",
           "msa_plan_export", "msa_workspace_bytes", "msa_forward", "msa_forward_host",
           "msa_last_launch_count", "msa_set_timing", "msa_get_timing", "msa_strerror", "msa_last_cuda_error", "msa_version",
           "msa_append_plan_create", "msa_append_plan_destroy", "msa_kv_append",
           "msa_plan_create_writeback", "msa_forward_writeback", "msa_forward_host_async", "msa_forward_host_wait",
           "msa_forward_static_ws", "msa_check_block_ids"]
EVICTOR_EXPORTS = ["msa_evictor_create", "msa_evictor_destroy", "msa_evictor_add", "msa_evictor_remove", "msa_evictor_evict",
                   "msa_evictor_evict_linear", "msa_evictor_set_lambda", "msa_evictor_size", "msa_evictor_weight"]


class MsaAppend(ctypes.Structure):
    _fields_ = [("row_off", ctypes.c_int64), ("len", ctypes.c_int32), ("block_off", ctypes.c_int32)]


class MsaEvictorConfig(ctypes.Structure):
    _fields_ = [("alpha", ctypes.c_double), ("beta", ctypes.c_double), ("tau0", ctypes.c_double),
                ("lambda_", ctypes.c_double), ("k5", ctypes.c_double), ("c0", ctypes.c_double)]


def _lib() -> ctypes.CDLL:
    global _LIB
    if _LIB is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -c 'import __graft_entry__ as g; "
                               "g.build()'` (there is no fallback path)")
        lib = ctypes.CDLL(LIB_PATH)
        vp, i32, i64, f32, sz = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_float, ctypes.c_size_t
        lib.msa_create.argtypes = [ctypes.POINTER(MsaConfig), ctypes.POINTER(vp)]
        lib.msa_destroy.argtypes = [vp]
        lib.msa_destroy.restype = None
        lib.msa_plan_create.argtypes = [vp, ctypes.POINTER(MsaRequest), i32, ctypes.POINTER(MsaSegment), i32,
                                        ctypes.POINTER(vp)]
        lib.msa_plan_destroy.argtypes = [vp]
        lib.msa_plan_destroy.restype = None
        lib.msa_plan_get_info.argtypes = [vp, ctypes.POINTER(MsaPlanInfo)]
        lib.msa_plan_export.argtypes = [vp, ctypes.c_int, vp, ctypes.POINTER(sz)]
        lib.msa_workspace_bytes.argtypes = [vp, ctypes.POINTER(sz)]
        lib.msa_forward.argtypes = [vp, vp, vp, i64, vp, vp, i64, vp, i64, vp, vp, i64, f32, vp, vp, vp, sz, vp]
        lib.msa_forward_host.argtypes = [vp, vp, vp, i64, vp, vp, i64, vp, i64, vp, vp, i64, f32, vp, vp, vp]
        lib.msa_forward_static_ws.argtypes = [vp, vp, vp, i64, vp, vp, i64, vp, i64, vp, vp, i64, f32, vp, vp, vp]
        lib.msa_forward_host_async.argtypes = [vp, vp, vp, i64, vp, vp, i64, vp, i64, vp, vp, i64, f32, vp, vp, vp, i32]
        lib.msa_forward_host_wait.argtypes = [vp, i32]
        lib.msa_check_block_ids.argtypes = [vp, vp, vp, vp, i64, i64, vp, vp]
        lib.msa_last_launch_count.argtypes = [vp]
        lib.msa_set_timing.argtypes = [vp, ctypes.c_int]
        lib.msa_get_timing.argtypes = [vp, ctypes.POINTER(i32), ctypes.POINTER(ctypes.c_double),
                                       ctypes.POINTER(ctypes.c_double)]
        for f in ("msa_strerror", "msa_last_cuda_error", "msa_version"):
            getattr(lib, f).restype = ctypes.c_char_p
        lib.msa_strerror.argtypes = [ctypes.c_int]
        lib.msa_append_plan_create.argtypes = [vp, ctypes.POINTER(MsaAppend), i32, ctypes.POINTER(vp)]
        lib.msa_append_plan_destroy.argtypes = [vp]
        lib.msa_append_plan_destroy.restype = None
        lib.msa_kv_append.argtypes = [vp, vp, vp, vp, i64, vp, vp, i64, vp, i64, vp]
        lib.msa_plan_create_writeback.argtypes = [vp, ctypes.POINTER(MsaRequest), i32, ctypes.POINTER(MsaSegment), i32,
                                                  ctypes.POINTER(MsaAppend), i32, ctypes.POINTER(vp)]
        lib.msa_forward_writeback.argtypes = [vp, vp, vp, i64, vp, vp, i64, vp, i64, vp, vp, i64, f32, vp, vp, vp, sz, vp]
        f64 = ctypes.c_double
        lib.msa_evictor_create.argtypes = [ctypes.POINTER(MsaEvictorConfig), ctypes.POINTER(vp)]
        lib.msa_evictor_destroy.argtypes = [vp]
        lib.msa_evictor_destroy.restype = None
        lib.msa_evictor_add.argtypes = [vp, i64, i64, f64]
        lib.msa_evictor_remove.argtypes = [vp, i64]
        lib.msa_evictor_evict.argtypes = [vp, f64, ctypes.POINTER(i64)]
        lib.msa_evictor_evict_linear.argtypes = [vp, f64, ctypes.POINTER(i64)]
        lib.msa_evictor_set_lambda.argtypes = [vp, f64]
        lib.msa_evictor_size.argtypes = [vp]
        lib.msa_evictor_size.restype = i64
        lib.msa_evictor_weight.argtypes = [vp, i64, f64]
        lib.msa_evictor_weight.restype = f64
        _LIB = lib
    return _LIB


def _check(status: int, where: str) -> None:
    if status != MSA_OK:
        raise MsaError(status, where)


def _dptr(t) -> Optional[int]:
    """Device/host pointer of a torch tensor or numpy array (None -> NULL)."""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        return t.ctypes.data
    return t.data_ptr()


def msa_version() -> str:
    return _lib().msa_version().decode()


def msa_create(num_q_heads: int, num_kv_heads: int, head_dim: int, q_to_kv_head=None, device: int = 0,
               block_size: int = 16, pool_format: int = MSA_POOL_BF16, k_scale=None, v_scale=None) -> ctypes.c_void_p:
    """pool_format = MSA_POOL_FP8_E4M3: the paged pool holds E4M3 codes; k_scale / v_scale float32 [Hkv] (powers of two)."""
    cfg = MsaConfig(num_q_heads, num_kv_heads, head_dim, block_size, None, device, pool_format, None, None)
    keep = None
    if q_to_kv_head is not None:
        keep = np.ascontiguousarray(q_to_kv_head, np.int32)
        cfg.q_to_kv_head = keep.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))
    keep_s = []
    for name, sc in (("k_scale", k_scale), ("v_scale", v_scale)):
        if sc is not None:
            arr = np.ascontiguousarray(sc, np.float32)
            keep_s.append(arr)
            setattr(cfg, name, arr.ctypes.data_as(ctypes.POINTER(ctypes.c_float)))
    h = ctypes.c_void_p()
    _check(_lib().msa_create(ctypes.byref(cfg), ctypes.byref(h)), "msa_create")
    return h


def msa_destroy(h) -> None:
    _lib().msa_destroy(h)


def make_descriptors(req: np.ndarray, seg_kind, seg_abs_start, seg_len, seg_block_off, seg_row_off):
    """numpy descriptor columns -> ctypes arrays of msa_request / msa_segment."""
    req = np.asarray(req, np.int32).reshape(-1, 5)
    R = (MsaRequest * max(1, req.shape[0]))()
    for i in range(req.shape[0]):
        R[i] = MsaRequest(*(int(x) for x in req[i]))
    n = len(seg_kind)
    S = (MsaSegment * max(1, n))()
    for i in range(n):
        S[i] = MsaSegment(int(seg_kind[i]), int(seg_abs_start[i]), int(seg_len[i]), int(seg_block_off[i]),
                          int(seg_row_off[i]))
    return R, req.shape[0], S, n


def msa_plan_create(h, requests, n_req: int, segments, n_seg: int) -> ctypes.c_void_p:
    p = ctypes.c_void_p()
    _check(_lib().msa_plan_create(h, requests, n_req, segments, n_seg, ctypes.byref(p)), "msa_plan_create")
    return p


def msa_plan_destroy(p) -> None:
    _lib().msa_plan_destroy(p)


def msa_plan_get_info(p) -> Dict[str, int]:
    info = MsaPlanInfo()
    _check(_lib().msa_plan_get_info(p, ctypes.byref(info)), "msa_plan_get_info")
    return {k: int(getattr(info, k)) for k, _ in MsaPlanInfo._fields_}


_EXPORT_DTYPES = {
    0: np.dtype([("src", "<i4"), ("abs_start", "<i4"), ("nvalid", "<i4"), ("paged", "<i4")]),
    1: np.dtype([("q_row0", "<i4"), ("n_tok", "<i4"), ("q_abs0", "<i4"), ("kvh", "<i4"), ("vb_begin", "<i4"),
                 ("vb_count", "<i4"), ("tile_begin", "<i4"), ("tile_end", "<i4"), ("partial_off", "<i4"),
                 ("mode", "<i4"), ("tile_info_begin", "<i4"), ("writeback", "<i4")]),
    2: np.dtype("<i4"),
    3: np.dtype([("q_row0", "<i4"), ("n_tok", "<i4"), ("kvh", "<i4"), ("n_partials", "<i4"),
                 ("first_off", "<i8"), ("stride", "<i8")]),
    4: np.dtype([("max_abs", "<i4"), ("ragged", "<i4")]),
    5: np.dtype("<i4"),
    6: np.dtype("<i4"),
    7: np.dtype("<i4"),
}


def msa_plan_export(p, which: int) -> np.ndarray:
    n = ctypes.c_size_t(0)
    _check(_lib().msa_plan_export(p, which, None, ctypes.byref(n)), "msa_plan_export")
    dt = _EXPORT_DTYPES[which]
    out = np.zeros(n.value // dt.itemsize, dt)
    if n.value:
        _check(_lib().msa_plan_export(p, which, out.ctypes.data, ctypes.byref(n)), "msa_plan_export")
    return out


def msa_workspace_bytes(p) -> int:
    n = ctypes.c_size_t(0)
    _check(_lib().msa_workspace_bytes(p, ctypes.byref(n)), "msa_workspace_bytes")
    return int(n.value)


def msa_forward(h, p, q, pool_k, pool_v, block_table, contig_k, contig_v, softmax_scale: float, o, lse,
                workspace=None, stream: Optional[int] = None) -> None:
    """q/pool/contig/o: bf16 CUDA tensors; block_table int32 CUDA; lse fp32 CUDA; workspace uint8 CUDA."""
    total_q = int(q.shape[0])
    num_blocks = 0 if pool_k is None else int(pool_k.shape[0])
    bt_len = 0 if block_table is None else int(block_table.numel())
    rows = 0 if contig_k is None else int(contig_k.shape[0])
    ws_bytes = 0 if workspace is None else int(workspace.numel() * workspace.element_size())
    _check(_lib().msa_forward(h, p, _dptr(q), total_q, _dptr(pool_k), _dptr(pool_v), num_blocks, _dptr(block_table),
                              bt_len, _dptr(contig_k), _dptr(contig_v), rows, ctypes.c_float(softmax_scale), _dptr(o),
                              _dptr(lse), _dptr(workspace), ws_bytes, stream), "msa_forward")


def msa_forward_static_ws(h, p, q, pool_k, pool_v, block_table, contig_k, contig_v, softmax_scale: float, o, lse,
                          stream: Optional[int] = None) -> None:
    """msa_forward for a caller that cannot allocate the workspace (all HBM already belongs to its KV pool, or cudaMalloc is
    off limits while steps are in flight): the library's built-in MSA_STATIC_WS_BYTES array is the workspace.  Raises
    MsaError(MSA_ERR_STATIC_WS) when the plan needs more.  One array per device: calls that overlap on the GPU race."""
    total_q = int(q.shape[0])
    num_blocks = 0 if pool_k is None else int(pool_k.shape[0])
    bt_len = 0 if block_table is None else int(block_table.numel())
    rows = 0 if contig_k is None else int(contig_k.shape[0])
    _check(_lib().msa_forward_static_ws(h, p, _dptr(q), total_q, _dptr(pool_k), _dptr(pool_v), num_blocks,
                                        _dptr(block_table), bt_len, _dptr(contig_k), _dptr(contig_v), rows,
                                        ctypes.c_float(softmax_scale), _dptr(o), _dptr(lse), stream),
           "msa_forward_static_ws")


def msa_forward_host(h, p, q_host, pool_k, pool_v, block_table_host, contig_k_host, contig_v_host,
                     softmax_scale: float, o_host, lse_host, stream: Optional[int] = None) -> None:
    """Host (ideally pinned) q / block table / arena / o / lse; the paged pool stays on the device."""
    total_q = int(q_host.shape[0])
    num_blocks = 0 if pool_k is None else int(pool_k.shape[0])
    bt_len = 0 if block_table_host is None else int(block_table_host.numel())
    rows = 0 if contig_k_host is None else int(contig_k_host.shape[0])
    _check(_lib().msa_forward_host(h, p, _dptr(q_host), total_q, _dptr(pool_k), _dptr(pool_v), num_blocks,
                                   _dptr(block_table_host), bt_len, _dptr(contig_k_host), _dptr(contig_v_host), rows,
                                   ctypes.c_float(softmax_scale), _dptr(o_host), _dptr(lse_host), stream),
           "msa_forward_host")


def msa_forward_host_async(h, p, q_host, pool_k, pool_v, block_table_host, contig_k_host, contig_v_host,
                           softmax_scale: float, o_host, lse_host, stream: Optional[int] = None, slot: int = 0) -> None:
    """msa_forward_host without the wait (two slots; results valid after msa_forward_host_wait(h, slot))."""
    total_q = int(q_host.shape[0])
    num_blocks = 0 if pool_k is None else int(pool_k.shape[0])
    bt_len = 0 if block_table_host is None else int(block_table_host.numel())
    rows = 0 if contig_k_host is None else int(contig_k_host.shape[0])
    _check(_lib().msa_forward_host_async(h, p, _dptr(q_host), total_q, _dptr(pool_k), _dptr(pool_v), num_blocks,
                                         _dptr(block_table_host), bt_len, _dptr(contig_k_host), _dptr(contig_v_host), rows,
                                         ctypes.c_float(softmax_scale), _dptr(o_host), _dptr(lse_host), stream, slot),
           "msa_forward_host_async")


def msa_forward_host_wait(h, slot: int = 0) -> None:
    _check(_lib().msa_forward_host_wait(h, slot), "msa_forward_host_wait")


def msa_check_block_ids(h, plan, append_plan, block_table, num_blocks: int, flag, stream: Optional[int] = None) -> None:
    """Debug check: flag (int32 CUDA tensor, 1 element) <- smallest block-table index the plan(s) refer to whose id is outside
    [0, num_blocks), or -1.  Asynchronous on `stream`."""
    _check(_lib().msa_check_block_ids(h, plan, append_plan, _dptr(block_table), int(block_table.numel()), int(num_blocks),
                                      _dptr(flag), stream), "msa_check_block_ids")


def msa_last_launch_count(h) -> int:
    return int(_lib().msa_last_launch_count(h))


def msa_set_timing(h, max_steps: int) -> None:
    _check(_lib().msa_set_timing(h, max_steps), "msa_set_timing")


def msa_get_timing(h) -> Tuple[int, float, float]:
    """(steps recorded, average forward-kernel ms, average merge-kernel ms)."""
    n, a, b = ctypes.c_int32(0), ctypes.c_double(0), ctypes.c_double(0)
    _check(_lib().msa_get_timing(h, ctypes.byref(n), ctypes.byref(a), ctypes.byref(b)), "msa_get_timing")
    return int(n.value), float(a.value), float(b.value)


# --------------------------------------------------------------------------- convenience
class MsaSession:
    """Handle + plan + output/workspace buffers for one problem (marshalling only)."""

    def __init__(self, problem, device: int = 0):
        import torch
        self.problem = p = problem
        kv8 = getattr(p, "k_scale", None) is not None       # fp8 (E4M3) paged pool
        self.h = msa_create(p.Hq, p.Hkv, p.D, p.q_to_kv, device=device,
                            pool_format=MSA_POOL_FP8_E4M3 if kv8 else MSA_POOL_BF16,
                            k_scale=p.k_scale if kv8 else None, v_scale=p.v_scale if kv8 else None)
        R, n_req, S, n_seg = make_descriptors(p.req, p.seg_kind, p.seg_abs_start, p.seg_len, p.seg_block_off,
                                              p.seg_row_off)
        self.plan = msa_plan_create(self.h, R, n_req, S, n_seg)
        self.info = msa_plan_get_info(self.plan)
        dev = torch.device("cuda", device)
        self.o = torch.zeros((p.total_q, p.Hq, p.D), dtype=torch.bfloat16, device=dev)
        self.lse = torch.zeros((p.total_q, p.Hq), dtype=torch.float32, device=dev)
        nb = msa_workspace_bytes(self.plan)
        self.workspace = torch.empty(max(nb, 16), dtype=torch.uint8, device=dev) if nb else None

    def forward(self, stream: Optional[int] = None) -> Tuple["object", "object"]:
        import torch
        p = self.problem
        if stream is None:
            stream = torch.cuda.current_stream().cuda_stream
        msa_forward(self.h, self.plan, p.q, p.pool_k, p.pool_v, p.block_table, p.contig_k, p.contig_v, p.scale,
                    self.o, self.lse, self.workspace, stream)
        return self.o, self.lse

    def close(self) -> None:
        if self.plan is not None:
            msa_plan_destroy(self.plan)
            self.plan = None
        if self.h is not None:
            msa_destroy(self.h)
            self.h = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()



# --------------------------------------------------------------------------- KV write-back
def msa_append_plan_create(h, jobs):
    """jobs: iterable of (row_off, len, block_off)."""
    jobs = list(jobs)
    arr = (MsaAppend * max(1, len(jobs)))()
    for i, (row_off, n, block_off) in enumerate(jobs):
        arr[i] = MsaAppend(int(row_off), int(n), int(block_off))
    ap = ctypes.c_void_p()
    _check(_lib().msa_append_plan_create(h, arr, len(jobs), ctypes.byref(ap)), "msa_append_plan_create")
    return ap


def msa_plan_create_writeback(h, requests, n_req: int, segments, n_seg: int, jobs) -> ctypes.c_void_p:
    """jobs: iterable of (row_off, len, block_off), as in msa_append_plan_create."""
    jobs = list(jobs)
    arr = (MsaAppend * max(1, len(jobs)))()
    for i, (row_off, n, block_off) in enumerate(jobs):
        arr[i] = MsaAppend(int(row_off), int(n), int(block_off))
    p = ctypes.c_void_p()
    _check(_lib().msa_plan_create_writeback(h, requests, n_req, segments, n_seg, arr, len(jobs), ctypes.byref(p)),
           "msa_plan_create_writeback")
    return p


def msa_forward_writeback(h, p, q, pool_k, pool_v, block_table, contig_k, contig_v, softmax_scale: float, o, lse,
                          workspace=None, stream: Optional[int] = None) -> None:
    """msa_forward that also writes the plan's write-back jobs into pool_k / pool_v (same launch)."""
    total_q = int(q.shape[0])
    num_blocks = 0 if pool_k is None else int(pool_k.shape[0])
    bt_len = 0 if block_table is None else int(block_table.numel())
    rows = 0 if contig_k is None else int(contig_k.shape[0])
    ws_bytes = 0 if workspace is None else int(workspace.numel() * workspace.element_size())
    _check(_lib().msa_forward_writeback(h, p, _dptr(q), total_q, _dptr(pool_k), _dptr(pool_v), num_blocks,
                                        _dptr(block_table), bt_len, _dptr(contig_k), _dptr(contig_v), rows,
                                        ctypes.c_float(softmax_scale), _dptr(o), _dptr(lse), _dptr(workspace), ws_bytes,
                                        stream), "msa_forward_writeback")


def msa_append_plan_destroy(ap) -> None:
    _lib().msa_append_plan_destroy(ap)


def msa_kv_append(h, ap, contig_k, contig_v, pool_k, pool_v, block_table, stream: Optional[int] = None) -> None:
    """Arena rows -> paged cache blocks (bf16 CUDA tensors; block_table int32 CUDA); asynchronous on `stream`."""
    rows = 0 if contig_k is None else int(contig_k.shape[0])
    nb = 0 if pool_k is None else int(pool_k.shape[0])
    bt_len = 0 if block_table is None else int(block_table.numel())
    _check(_lib().msa_kv_append(h, ap, _dptr(contig_k), _dptr(contig_v), rows, _dptr(pool_k), _dptr(pool_v), nb,
                                _dptr(block_table), bt_len, stream), "msa_kv_append")


# --------------------------------------------------------------------------- block evictor (include/msa_evictor.h)
class MsaEvictor:
    """ctypes view of the C++ evictor (Algorithm 1): argument marshalling only."""

    def __init__(self, alpha: float, beta: float, tau0: float, k5: float, c0: float, lambda_: float = 1.0):
        cfg = MsaEvictorConfig(alpha, beta, tau0, lambda_, k5, c0)
        self._h = ctypes.c_void_p()
        _check(_lib().msa_evictor_create(ctypes.byref(cfg), ctypes.byref(self._h)), "msa_evictor_create")

    def add(self, block_id: int, position: int, last_access: float) -> None:
        _check(_lib().msa_evictor_add(self._h, block_id, position, last_access), "msa_evictor_add")

    def remove(self, block_id: int) -> None:
        _check(_lib().msa_evictor_remove(self._h, block_id), "msa_evictor_remove")

    def evict(self, t_now: float, linear: bool = False) -> int:
        out = ctypes.c_int64(0)
        fn = _lib().msa_evictor_evict_linear if linear else _lib().msa_evictor_evict
        _check(fn(self._h, t_now, ctypes.byref(out)), "msa_evictor_evict")
        return int(out.value)

    def set_lambda(self, lambda_: float) -> None:
        _check(_lib().msa_evictor_set_lambda(self._h, lambda_), "msa_evictor_set_lambda")

    def weight(self, block_id: int, t_now: float) -> float:
        return float(_lib().msa_evictor_weight(self._h, block_id, t_now))

    def __len__(self) -> int:
        return int(_lib().msa_evictor_size(self._h))

    def close(self) -> None:
        if self._h:
            _lib().msa_evictor_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
