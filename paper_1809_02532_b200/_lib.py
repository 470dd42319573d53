"""ctypes loader of libtfa.so.  There is no fallback: a missing library is an error."""
from __future__ import annotations

import ctypes as C
import os

NEQ = 18
BLOCK = NEQ * NEQ
HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libtfa.so")


class TfaError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libtfa error {code}: {msg}")
        self.code = code


class Physics(C.Structure):
    """Mirror of ``tfa_physics`` (include/tfa.h)."""
    _fields_ = [("gamma_gas", C.c_double), ("mass_ratio", C.c_double), ("c", C.c_double),
                ("gamma_psi", C.c_double), ("chi_phi", C.c_double), ("rusanov_alpha", C.c_double)]


class Numerics(C.Structure):
    """Mirror of ``tfa_numerics`` (include/tfa.h)."""
    _fields_ = [("fd_delta", C.c_double), ("fd_ref", C.c_double * NEQ), ("venkat_K", C.c_double),
                ("lsq_weight_power", C.c_double), ("ausm_Kp", C.c_double), ("ausm_Ku", C.c_double),
                ("ausm_sigma", C.c_double), ("ausm_beta", C.c_double), ("ausm_Minf", C.c_double * 2),
                ("term_mask", C.c_int32), ("pad_", C.c_int32)]


# every symbol include/tfa.h declares: name -> (restype, argtypes)
_vp, _i64, _dbl, _int = C.c_void_p, C.c_int64, C.c_double, C.c_int
SYMBOLS = {
    "tfa_mesh_create": (_int, [C.POINTER(_vp), _i64, _vp, _i64, _vp, _vp, _vp]),
    "tfa_mesh_create_poly": (_int, [C.POINTER(_vp), _i64, _vp, _i64, _vp, _vp, _vp, _vp]),
    "tfa_mesh_info": (_int, [_vp, C.POINTER(C.c_int32), C.POINTER(_i64)]),
    "tfa_mesh_set_bc": (_int, [_vp, _vp, _vp]),
    "tfa_mesh_reorder": (_int, [_vp, _int, _vp, _vp]),
    "tfa_mesh_sizes": (_int, [_vp] + [C.POINTER(_i64)] * 4),
    "tfa_mesh_get": (_int, [_vp, _int, _vp, _i64]),
    "tfa_mesh_device_ptr": (_vp, [_vp, _int]),
    "tfa_mesh_destroy": (None, [_vp]),
    "tfa_default_physics": (None, [C.POINTER(Physics)]),
    "tfa_default_numerics": (None, [C.POINTER(Numerics), C.POINTER(Physics)]),
    "tfa_ctx_create": (_int, [C.POINTER(_vp)]),
    "tfa_set_physics": (_int, [_vp, C.POINTER(Physics)]),
    "tfa_set_numerics": (_int, [_vp, C.POINTER(Numerics)]),
    "tfa_set_ghost_states": (_int, [_vp, _vp, _i64]),
    "tfa_ctx_destroy": (None, [_vp]),
    "tfa_gradients": (_int, [_vp, _vp, _vp, _vp, _vp, _vp]),
    "tfa_assemble": (_int, [_vp, _vp, _vp, _vp, _vp, _dbl, _vp, _vp, _vp]),
    "tfa_assemble_host": (_int, [_vp, _vp, _vp, _vp, _vp, _dbl, _vp, _vp, _vp]),
    "tfa_assemble_packed": (_int, [_vp, _vp, _vp, _vp, _vp, _dbl, _vp, _vp, _vp, _vp]),
    "tfa_packed_to_bsr": (_int, [_vp, _vp, _vp, _vp, _vp]),
    "tfa_packed_spmv": (_int, [_vp, _vp, _vp, _vp, _vp, _vp]),
    "tfa_block_jacobi_packed": (_int, [_vp, _vp, _vp, _vp, _vp]),
    "tfa_gmres_packed": (_int, [_vp, _vp, _vp, _vp, _vp, _vp, _vp, _int, _int, _dbl, C.POINTER(C.c_double), _vp]),
    "tfa_to_f32": (_int, [_vp, _vp, _i64, _vp]),
    "tfa_packed_to_f32": (_int, [_vp, _vp, _vp, _vp, _vp, _vp]),
    "tfa_gmres_packed_f32": (_int, [_vp] * 9 + [_int, _int, _dbl, C.POINTER(C.c_double), _vp]),
    "tfa_assemble_gradient": (_int, [_vp, _vp, _vp, _vp]),
    "tfa_assemble_faces": (_int, [_vp, _vp, _vp, _vp, _vp, _dbl, _vp, _vp, _vp]),
    "tfa_face_states": (_vp, [_vp]),
    "tfa_assemble_faces_packed": (_int, [_vp, _vp, _vp, _vp, _vp, _dbl, _vp, _vp, _vp, _vp]),
    "tfa_face_states_static": (_int, [_vp, _vp, _vp, _vp, _vp]),
    "tfa_partition_create": (_int, [C.POINTER(_vp), _i64, _int, _vp, _vp, _vp, _int, _int]),
    "tfa_partition_destroy": (None, [_vp]),
    "tfa_partition_sizes": (_int, [_vp] + [C.POINTER(_i64)] * 4),
    "tfa_partition_count": (_i64, [_vp, _int, _int]),
    "tfa_partition_get": (_int, [_vp, _int, _int, _vp, _i64]),
    "tfa_shard_create": (_int, [C.POINTER(_vp), _vp, _int, _int, _vp]),
    "tfa_shard_destroy": (None, [_vp]),
    "tfa_shard_mesh": (_vp, [_vp]),
    "tfa_shard_partition": (_vp, [_vp]),
    "tfa_shard_info": (_int, [_vp, C.POINTER(_i64), C.POINTER(_i64)]),
    "tfa_shard_bface_global": (_int, [_vp, _vp, _i64]),
    "tfa_shard_pack": (_int, [_vp, _int, _int, _vp, _vp, _vp]),
    "tfa_shard_unpack": (_int, [_vp, _int, _int, _vp, _vp, _vp]),
    "tfa_check": (_int, [_vp, _vp]),
    "tfa_probe_dfma": (_int, [_int, _int, _vp, _vp]),
    "tfa_probe_copy": (_int, [_vp, _vp, _i64, _vp]),
    "tfa_probe_math": (_int, [_vp, _vp, _vp, _i64, _vp]),
    "tfa_bsr_spmv": (_int, [_vp, _vp, _vp, _vp, _vp]),
    "tfa_block_jacobi": (_int, [_vp, _vp, _vp, _vp, _vp]),
    "tfa_gmres": (_int, [_vp, _vp, _vp, _vp, _vp, _vp, _int, _int, _dbl, C.POINTER(C.c_double), _vp]),
    "tfa_implicit_step": (_int, [_vp, _vp, _vp, _vp, _vp, _dbl, _vp, _vp, _vp, _vp, _int, _dbl, _int, _int, _dbl, _int,
                                 C.POINTER(C.c_double), _vp]),
    "tfa_jvp": (_int, [_vp, _vp, _vp, _vp, _vp, _dbl, _vp, _vp, _dbl, _vp]),
    "tfa_gmres_jfnk": (_int, [_vp, _vp, _vp, _vp, _vp, _dbl, _vp, _vp, _vp, _int, _int, _dbl, C.POINTER(C.c_double), _vp]),
    "tfa_timing_enable": (_int, [_vp, _int]),
    "tfa_timing_read": (_int, [_vp, C.POINTER(C.c_double), C.POINTER(_int)]),
    "tfa_launches_per_assemble": (_int, [_vp]),
    "tfa_last_error": (C.c_char_p, []),
    "tfa_version": (C.c_char_p, []),
}

_lib = None


def load():
    """Load libtfa.so (building is the job of ``paper_1809_02532_b200.build``)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_1809_02532_b200.build` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    for name, (res, args) in SYMBOLS.items():
        fn = getattr(lib, name)     # AttributeError if the ABI and the header disagree
        fn.restype = res
        fn.argtypes = args
    _lib = lib
    return lib


def check(rc: int):
    if rc != 0:
        raise TfaError(rc, load().tfa_last_error().decode())
