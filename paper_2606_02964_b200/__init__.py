"""B200-native Multi-Segment Attention (MSA): hand-written sm_100a kernels behind a C ABI.

``include/msa.h`` is the boundary; this package holds the CUDA sources (``csrc/``), the
in-tree build helper and a ctypes binding with the same names.  No CPU fallback exists.
"""
from .binding import (  # noqa: F401
    MSA_OK, MSA_ERR_INVALID_ARG, MSA_ERR_UNSUPPORTED, MSA_ERR_OVERLAP, MSA_ERR_UNSORTED,
    MSA_ERR_OUT_OF_RANGE, MSA_ERR_MISALIGNED, MSA_ERR_WORKSPACE, MSA_ERR_CUDA, MSA_ERR_NO_DEVICE,
    MSA_ERR_STATIC_WS, MSA_STATIC_WS_BYTES, msa_forward_static_ws, msa_check_block_ids,
    MSA_SEG_PAGED, MSA_SEG_CONTIG, MSA_SEG_SELF, MSA_POOL_BF16, MSA_POOL_FP8_E4M3,
    MsaError, MsaSession, MsaEvictor, make_descriptors,
    msa_create, msa_destroy, msa_plan_create, msa_plan_destroy, msa_plan_get_info, msa_plan_export,
    msa_workspace_bytes, msa_forward, msa_forward_host, msa_forward_host_async, msa_forward_host_wait, msa_append_plan_create, msa_append_plan_destroy, msa_kv_append, msa_plan_create_writeback, msa_forward_writeback, msa_last_launch_count, msa_set_timing, msa_get_timing, msa_version,
)
from ._build import build, LIB_PATH  # noqa: F401
