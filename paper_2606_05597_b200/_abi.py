"""ctypes mirror of include/awr.h and the loader of libawr.so.

Argument marshalling only: every step of the path runs in the CUDA kernels behind the C ABI.
There is no CPU or other-architecture fallback: if the library cannot be built / loaded the
import of any entry point raises.
"""
from __future__ import annotations

import ctypes as C
import os
import threading

from . import build as _build

# ---- enums (include/awr.h)
AWR_OK = 0
AWR_ERR_NULL, AWR_ERR_SHAPE, AWR_ERR_DTYPE, AWR_ERR_ALIGN = -1, -2, -3, -4
AWR_ERR_PARAM, AWR_ERR_WORKSPACE, AWR_ERR_ARCH, AWR_ERR_CUDA = -5, -6, -7, -8
AWR_ERR_STATIC_LIMIT = -9
STATIC_WS_BYTES = 1 << 20
DTYPE_BF16, DTYPE_F32 = 0, 1
NORM_CONST_K, NORM_PER_TRAJ = 0, 1
FLAG_SAMPLE_STD = 1
FLAG_SUCCESS_FILTER = 2
FLAG_COUPLED = 4
FLAG_SKIP_UNIFORM = 8
W_K_BY_V, W_V_BY_K = 0, 1
KERNEL_AUTO, KERNEL_GENERIC, KERNEL_CLUSTER, KERNEL_CLUSTER_RF, KERNEL_CLUSTER_RF4 = 0, 1, 2, 3, 4
KERNEL_HEAD_1CTA, KERNEL_HEAD_2CTA, KERNEL_HEAD_2CTA_STORED = 5, 6, 7
KERNEL_FWD_STREAM = 8
KERNEL_HEAD_2CTA_E16 = 9
KERNEL_CLUSTER_RFS = 10
KERNEL_HEAD_2CTA_ROWREF = 11
KERNEL_CLUSTER_RFS_LATE = 12
ERRBIT_STEP_OFF, ERRBIT_TRAJ_OFF, ERRBIT_GROUP_OFF, ERRBIT_TARGET_RANGE = 1, 2, 4, 8

_vp = C.c_void_p


class awr_batch(C.Structure):
    _fields_ = [("n_tok", C.c_int64), ("V", C.c_int64), ("ld", C.c_int64),
                ("logits", _vp), ("target_ids", _vp), ("behave_lp", _vp), ("prox_lp", _vp),
                ("step_off", _vp), ("traj_off", _vp), ("group_off", _vp), ("rewards", _vp),
                ("n_steps", C.c_int32), ("n_traj", C.c_int32), ("n_groups", C.c_int32),
                ("logits_dtype", C.c_int32)]


class awr_params(C.Structure):
    _fields_ = [("k_norm", C.c_float), ("clip_eps", C.c_float), ("stale_cap", C.c_float),
                ("loss_scale", C.c_float), ("dual_clip_c", C.c_float),
                ("normalizer", C.c_int32), ("flags", C.c_uint32), ("kernel", C.c_int32)]


class awr_outputs(C.Structure):
    _fields_ = [("loss", _vp), ("dlogits", _vp), ("token_lp", _vp), ("clip_count", _vp),
                ("adv", _vp), ("tok_traj", _vp), ("target_logit", _vp), ("tok_term", _vp),
                ("tok_coef", _vp), ("err_word", _vp), ("dual_clip_count", _vp),
                ("token_entropy", _vp), ("ev_row_begin", _vp), ("ev_row_end", _vp)]


class awr_head_batch(C.Structure):
    _fields_ = [("n_tok", C.c_int64), ("V", C.c_int64), ("K", C.c_int64),
                ("hidden", _vp), ("w_head", _vp), ("target_ids", _vp), ("behave_lp", _vp),
                ("prox_lp", _vp), ("step_off", _vp), ("traj_off", _vp), ("group_off", _vp),
                ("rewards", _vp),
                ("n_steps", C.c_int32), ("n_traj", C.c_int32), ("n_groups", C.c_int32),
                ("w_layout", C.c_int32)]


class awr_head_outputs(C.Structure):
    _fields_ = [("loss", _vp), ("dhidden", _vp), ("dw_head", _vp), ("token_lp", _vp),
                ("clip_count", _vp), ("adv", _vp), ("tok_traj", _vp), ("tok_term", _vp),
                ("tok_coef", _vp), ("err_word", _vp), ("dual_clip_count", _vp),
                ("token_entropy", _vp)]


# name -> (restype, argtypes): every symbol include/awr.h declares
SYMBOLS = {
    "awr_loss_fwd_bwd": (C.c_int, [C.POINTER(awr_batch), C.POINTER(awr_params),
                                   C.POINTER(awr_outputs), _vp, C.c_size_t, _vp]),
    "awr_loss_fwd": (C.c_int, [C.POINTER(awr_batch), C.POINTER(awr_params),
                               C.POINTER(awr_outputs), _vp, C.c_size_t, _vp]),
    "awr_loss_fwd_bwd_static": (C.c_int, [C.POINTER(awr_batch), C.POINTER(awr_params),
                                          C.POINTER(awr_outputs), _vp]),
    "awr_group_advantage": (C.c_int, [_vp, _vp, C.c_int32, C.c_int32, C.c_uint32, _vp, _vp]),
    "awr_workspace_bytes": (C.c_size_t, [C.c_int64, C.c_int64, C.c_int32, C.c_int32, C.c_int32]),
    "awr_loss_fwd_bwd_host": (C.c_int, [C.POINTER(awr_batch), C.POINTER(awr_params),
                                        C.POINTER(awr_outputs), _vp, C.c_size_t, _vp]),
    "awr_host_workspace_bytes": (C.c_size_t, [C.c_int64, C.c_int64, C.c_int64, C.c_int32,
                                              C.c_int32, C.c_int32, C.c_int32]),
    "awr_loss_fwd_bwd_fused_head": (C.c_int, [C.POINTER(awr_head_batch), C.POINTER(awr_params),
                                              C.POINTER(awr_head_outputs), _vp, C.c_size_t, _vp]),
    "awr_head_workspace_bytes": (C.c_size_t, [C.c_int64, C.c_int64, C.c_int64, C.c_int32,
                                              C.c_int32, C.c_int32, C.c_int32]),
    "awr_loss_fwd_bwd_fused_head_host": (C.c_int, [C.POINTER(awr_head_batch), C.POINTER(awr_params),
                                                   C.POINTER(awr_head_outputs), _vp, C.c_size_t, _vp]),
    "awr_head_host_workspace_bytes": (C.c_size_t, [C.c_int64, C.c_int64, C.c_int64, C.c_int32,
                                                   C.c_int32, C.c_int32, C.c_int32]),
    "awr_head_launches_per_call": (C.c_int, [C.c_int64, C.c_int64, C.c_int64, C.c_int32]),
    "awr_gemm_bf16": (C.c_int, [_vp, C.c_int32, C.c_int64, _vp, C.c_int32, C.c_int64, C.c_int64,
                                C.c_int64, C.c_int64, _vp, C.c_int64, C.c_int32, _vp]),
    "awr_status_string": (C.c_char_p, [C.c_int]),
    "awr_version": (C.c_int, []),
    "awr_select_kernel": (C.c_int, [C.c_int64, C.c_int64, C.c_int32]),
    "awr_launches_per_call": (C.c_int, []),
}

_lock = threading.Lock()
_lib = None


def lib_path() -> str:
    return _build.LIB


def load():
    """Build (if stale) and load libawr.so; raises if that is impossible - no fallback."""
    global _lib
    with _lock:
        if _lib is not None:
            return _lib
        path = _build.build()
        if not os.path.exists(path):
            raise RuntimeError("libawr.so is missing and could not be built: " + path)
        lib = C.CDLL(path)
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(lib, name)          # AttributeError if the symbol is not exported
            fn.restype = res
            fn.argtypes = args
        _lib = lib
        return lib


class AwrError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        msg = load().awr_status_string(status).decode()
        super().__init__("%s failed: %s (%d)" % (where, msg, status))


def check(status: int, where: str) -> None:
    if status != AWR_OK:
        raise AwrError(status, where)
