"""ctypes loader for libqtt_b200.so and the C-ABI prototypes of include/qtt.h / include/qtt_diag.h.

No arithmetic here.  The library is built in-tree by ``python -m paper_2406_17823_b200.build``;
if it is missing, loading FAILS LOUDLY (there is no CPU fallback).
"""
from __future__ import annotations

import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libqtt_b200.so")

QTT_OK = 0
STATUS_NAMES = {
    0: "QTT_OK", -1: "QTT_INVALID_ARG", -2: "QTT_SHAPE_MISMATCH", -3: "QTT_CAPACITY", -4: "QTT_CUDA",
    -5: "QTT_NUMERIC",
}

ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)
RELEASE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)

_P = C.c_void_p
_PP = C.POINTER(C.c_void_p)
_DP = C.POINTER(C.c_double)
_IP = C.POINTER(C.c_int)
_DPP = C.POINTER(_DP)

# name -> (restype, argtypes); every symbol include/*.h declares
PROTOTYPES = {
    # include/qtt.h
    "qtt_ctx_create": (C.c_int, [_PP, C.c_int, _P, ALLOC_FN, RELEASE_FN, _P, C.c_size_t]),
    "qtt_ctx_destroy": (None, [_P]),
    "qtt_last_error": (C.c_char_p, [_P]),
    "qtt_ctx_set_chi_work": (C.c_int, [_P, C.c_int]),
    "qtt_ctx_set_materialize_limit": (C.c_int, [_P, C.c_size_t]),
    "qtt_ctx_set_graphs": (C.c_int, [_P, C.c_int]),
    "qtt_ctx_set_convection": (C.c_int, [_P, C.c_int]),
    "qtt_ctx_set_phys_dim": (C.c_int, [_P, C.c_int]),
    "qtt_ctx_phys_dim": (C.c_int, [_P]),
    "qtt_rk4_step3": (C.c_int, [_P, _PP, _PP, _P, C.c_double, C.c_double, C.c_int, C.c_double]),
    "qtt_ctx_set_product_compression": (C.c_int, [_P, C.c_int, C.c_ulonglong]),
    "qtt_ctx_jacobi_stats": (C.c_int, [_P, _IP, _IP]),
    "qtt_ctx_launch_count": (C.c_longlong, [_P]),
    "qtt_ctx_profile": (C.c_int, [_P, C.c_int]),
    "qtt_ctx_profile_report": (C.c_int, [_P, _DP, _DP, C.POINTER(C.c_longlong)]),
    "qtt_mps_from_dense": (C.c_int, [_P, _P, C.c_int, C.c_int, C.c_double, _PP]),
    "qtt_mps_from_cores": (C.c_int, [_P, C.c_int, _IP, _DPP, _PP]),
    "qtt_to_dense": (C.c_int, [_P, _P, _P]),
    "qtt_mpo_create": (C.c_int, [_P, C.c_int, _IP, _DPP, _PP]),
    "qtt_mpo_central_difference": (C.c_int, [_P, C.c_int, C.c_int, C.c_double, _PP]),
    "qtt_mpo_stencil": (C.c_int, [_P, C.c_int, C.c_int, C.c_int, _DP, _PP]),
    "qtt_mpo_laplacian": (C.c_int, [_P, C.c_int, C.c_double, _PP]),
    "qtt_mpo_free": (None, [_P]),
    "qtt_apply_mpo": (C.c_int, [_P, _P, _P, _PP]),
    "qtt_hadamard": (C.c_int, [_P, _P, _P, _PP]),
    "qtt_axpy": (C.c_int, [_P, C.c_double, _P, _P]),
    "qtt_round": (C.c_int, [_P, _P, C.c_int, C.c_double]),
    "qtt_round_ex": (C.c_int, [_P, _P, C.c_int, C.c_double, C.c_int]),
    "qtt_mps_core_ptr": (C.c_int, [_P, _P, C.c_int, C.POINTER(C.c_void_p)]),
    "qtt_round_batch": (C.c_int, [_P, C.c_int, _PP, C.c_int, C.c_double]),
    "qtt_rk4_step": (C.c_int, [_P, _PP, _P, _P, _P, C.c_double, C.c_double, C.c_int, C.c_double]),
    "qtt_mps_num_sites": (C.c_int, [_P]),
    "qtt_mps_bonds": (C.c_int, [_P, _IP]),
    "qtt_mps_get_core": (C.c_int, [_P, _P, C.c_int, _DP]),
    "qtt_mps_dot": (C.c_int, [_P, _P, _P, _DP]),
    "qtt_mps_norm": (C.c_int, [_P, _P, _DP]),
    "qtt_mps_schmidt": (C.c_int, [_P, _P, _DP, C.c_int, _IP]),
    "qtt_mps_fidelity": (C.c_int, [_P, _P, _P, _DP]),
    "qtt_mps_chi_eps": (C.c_int, [_P, _P, C.c_double, _IP, _IP]),
    "qtt_tke_spectrum": (C.c_int, [_P, _P, _P, _P, _P, C.c_int, _DP]),
    "qtt_variational_cost": (C.c_int, [_P, _PP, _PP, _PP, _P, _P, C.c_double, C.c_double, _DP]),
    "qtt_variational_stage": (C.c_int, [_P, _PP, _PP, _PP, _P, _P, C.c_double, C.c_double, C.c_int, C.c_double, C.c_int,
                                        C.c_double, _IP, C.POINTER(C.c_longlong), _IP]),
    "qtt_mps_clone": (C.c_int, [_P, _P, _PP]),
    "qtt_mps_free": (None, [_P]),
    # include/qtt_diag.h
    "qtt_diag_gemm": (C.c_int, [_P, _P, _P, _P, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_longlong,
                                C.c_longlong, C.c_longlong, C.c_double, C.c_double, C.c_int, C.c_longlong,
                                C.c_longlong, C.c_longlong]),
    "qtt_diag_lq": (C.c_int, [_P, _P, C.c_int, C.c_int, C.c_int, C.c_int, _P, _P]),
    "qtt_lq_noalloc": (C.c_int, [_P, _P, C.c_int, C.c_int, C.c_int, C.c_int, _P]),
    "qtt_diag_rowjacobi": (C.c_int, [_P, _P, C.c_int, C.c_int, C.c_int, C.c_int, _P]),
    "qtt_diag_rowjacobi_streamed": (C.c_int, [_P, _P, C.c_int, C.c_int, C.c_int, C.c_int, _P, _P]),
    "qtt_diag_svd_rows": (C.c_int, [_P, _P, C.c_int, C.c_int, C.c_int, C.c_int, _P, _P]),
    "qtt_diag_select": (C.c_int, [_P, _P, C.c_int, C.c_int, C.c_int, _P, C.c_int, _P, _P, C.c_int, C.c_double]),
    "qtt_diag_fp64_probe": (C.c_int, [_P, C.c_int, C.c_int, C.c_int, _DP]),
    "qtt_diag_profile_dump": (C.c_int, [C.c_char_p]),
}

_lib = None


def load() -> C.CDLL:
    """dlopen the in-tree library and attach the prototypes.  Raises if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(
            f"{LIB_PATH} is missing: build it with `python -m paper_2406_17823_b200.build` "
            "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    for name, (res, args) in PROTOTYPES.items():
        fn = getattr(lib, name)  # AttributeError if a declared symbol is not exported
        fn.restype = res
        fn.argtypes = args
    _lib = lib
    return lib
