"""ctypes front end of the fp64 CPU oracle (``msa_oracle.c``).

TEST INFRASTRUCTURE ONLY: importable from ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs, never from the product
package.  It does not import the product package either.

``forward(arrays, row_req, row_idx)`` takes the raw host arrays of a problem
(``workloads.MsaProblem.host_arrays()``): bf16 tensors as uint16, the block table, and
the request / segment descriptors -- i.e. exactly what the C-ABI library is given, not
its plan -- and returns (O fp64 [n,Hq,D], LSE fp64 [n,Hq]).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Dict, Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "msa_oracle.c")
_LIB = os.path.join(_HERE, "libmsa_oracle.so")
_lib: Optional[ctypes.CDLL] = None


def build(force: bool = False) -> str:
    """Compile msa_oracle.c with gcc (-O2, OpenMP, no fast-math) next to the source."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.run(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-o", tmp, _SRC, "-lm"],
                       check=True)
        os.replace(tmp, _LIB)
    return _LIB


def _load() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.msa_oracle_forward.restype = ctypes.c_int
        _lib.msa_oracle_forward_kv8.restype = ctypes.c_int
        _lib.msa_oracle_e4m3_to_double.restype = ctypes.c_double
        _lib.msa_oracle_e4m3_to_double.argtypes = [ctypes.c_uint8]
        _lib.msa_oracle_num_threads.restype = ctypes.c_int
    return _lib


def num_threads() -> int:
    return int(_load().msa_oracle_num_threads())


def e4m3_to_double(code: int) -> float:
    """Value of one OCP FP8 E4M3 code (the oracle's own decoder, written from the format's definition)."""
    return float(_load().msa_oracle_e4m3_to_double(ctypes.c_uint8(int(code) & 0xff)))


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def forward(a: Dict[str, np.ndarray], Hq: int, Hkv: int, D: int, scale: float,
            row_req: np.ndarray, row_idx: np.ndarray) -> Tuple[np.ndarray, np.ndarray]:
    lib = _load()
    req = np.ascontiguousarray(a["req"], np.int32)
    cols = [np.ascontiguousarray(req[:, c]) for c in range(5)]
    row_req = np.ascontiguousarray(row_req, np.int32)
    row_idx = np.ascontiguousarray(row_idx, np.int32)
    n = int(row_req.shape[0])
    O = np.zeros((n, Hq, D), np.float64)
    LSE = np.zeros((n, Hq), np.float64)
    kv8 = a.get("k_scale") is not None      # fp8 (E4M3) paged pool: bytes + one fp32 scale per KV head
    pool_dt = np.uint8 if kv8 else np.uint16
    if kv8:
        assert a["pool_k"].dtype == np.uint8 and a["pool_v"].dtype == np.uint8
    keep = dict(
        q=np.ascontiguousarray(a["q"], np.uint16),
        pool_k=np.ascontiguousarray(a["pool_k"], pool_dt), pool_v=np.ascontiguousarray(a["pool_v"], pool_dt),
        bt=np.ascontiguousarray(a["block_table"], np.int32),
        ck=np.ascontiguousarray(a["contig_k"], np.uint16), cv=np.ascontiguousarray(a["contig_v"], np.uint16),
        sk=np.ascontiguousarray(a["seg_kind"], np.int32), sa=np.ascontiguousarray(a["seg_abs_start"], np.int32),
        sl=np.ascontiguousarray(a["seg_len"], np.int32), sb=np.ascontiguousarray(a["seg_block_off"], np.int32),
        sr=np.ascontiguousarray(a["seg_row_off"], np.int64),
        hm=None if a.get("q_to_kv") is None else np.ascontiguousarray(a["q_to_kv"], np.int32))
    scales = ()
    fn = lib.msa_oracle_forward
    if kv8:
        keep["ks"] = np.ascontiguousarray(a["k_scale"], np.float32)
        keep["vs"] = np.ascontiguousarray(a["v_scale"], np.float32)
        assert keep["ks"].shape == (Hkv,) and keep["vs"].shape == (Hkv,)
        scales = (_ptr(keep["ks"]), _ptr(keep["vs"]))
        fn = lib.msa_oracle_forward_kv8
    rc = fn(
        ctypes.c_int(Hq), ctypes.c_int(Hkv), ctypes.c_int(D), _ptr(keep["hm"]),
        _ptr(keep["q"]), _ptr(keep["pool_k"]), _ptr(keep["pool_v"]), *scales, _ptr(keep["bt"]),
        _ptr(keep["ck"]), _ptr(keep["cv"]),
        ctypes.c_int(req.shape[0]), _ptr(cols[0]), _ptr(cols[1]), _ptr(cols[2]), _ptr(cols[3]), _ptr(cols[4]),
        _ptr(keep["sk"]), _ptr(keep["sa"]), _ptr(keep["sl"]), _ptr(keep["sb"]), _ptr(keep["sr"]),
        ctypes.c_float(scale),
        ctypes.c_int64(n), _ptr(row_req), _ptr(row_idx), _ptr(O), _ptr(LSE))
    if rc != 0:
        raise RuntimeError(f"msa_oracle_forward failed: {rc}")
    return O, LSE


def forward_problem(p, row_req: Optional[np.ndarray] = None, row_idx: Optional[np.ndarray] = None,
                    arrays: Optional[Dict[str, np.ndarray]] = None) -> Tuple[np.ndarray, np.ndarray]:
    """Oracle over a ``workloads.MsaProblem`` (duck-typed; no import of the generator here).
    Default: every query row, in q-row order."""
    if row_req is None:
        row_req = np.concatenate([np.full(int(p.req[r, 1]), r, np.int32) for r in range(p.req.shape[0])])
        row_idx = np.concatenate([np.arange(int(p.req[r, 1]), dtype=np.int32) for r in range(p.req.shape[0])])
    if arrays is None:
        arrays = p.host_arrays(reqs=sorted(set(int(x) for x in row_req)))
    return forward(arrays, p.Hq, p.Hkv, p.D, p.scale, row_req, row_idx)
