"""ctypes loader of libb200sht.so (built in-tree by paper_2311_14670_b200/build.py).  No fallback: a missing or
unloadable library is an error."""
import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libb200sht.so")

SHT_MW, SHT_HEALPIX, SHT_MWSS, SHT_DH, SHT_GL = 0, 1, 2, 3, 4
SHT_F64, SHT_F32 = 0, 1
SHT_OPT_FOLD_ON, SHT_OPT_FOLD_OFF, SHT_OPT_INVSYM, SHT_OPT_TILE64, SHT_OPT_TILE128, SHT_OPT_ADJOINT, SHT_OPT_PRECOMPUTE, SHT_OPT_NO_INVSYM = 1, 2, 4, 8, 16, 32, 64, 128
SHT_OPT_NO_PAIR, SHT_OPT_GRAPH, SHT_OPT_NO_GRAPH, SHT_OPT_NO_SKIP = 256, 512, 1024, 2048
SHT_PEAK_DFMA, SHT_PEAK_DMMA, SHT_PEAK_FFMA, SHT_PEAK_FFMA2 = 0, 1, 2, 3
SHT_NOALLOC_SCRATCH_BYTES, SHT_NOALLOC_MAX_RINGS = 8 << 20, 128

# every symbol include/b200sht.h declares: name -> (restype, argtypes)
_vp, _i, _sz = C.c_void_p, C.c_int, C.c_size_t
SIGNATURES = {
    "sht_status_string": (C.c_char_p, [_i]),
    "sht_last_error": (C.c_char_p, []),
    "sht_plan_s2": (_i, [C.POINTER(_vp), _i, _i, _i, _i, _i, _i]),
    "sht_plan_so3": (_i, [C.POINTER(_vp), _i, _i, _i]),
    "sht_plan_so3_opts": (_i, [C.POINTER(_vp), _i, _i, _i, C.c_uint]),
    "so3_forward_adjoint_plan": (_i, [_vp, _vp, _vp, _vp]),
    "so3_inverse_adjoint_plan": (_i, [_vp, _vp, _vp, _vp]),
    "sht_plan_s2_batch": (_i, [C.POINTER(_vp), _i, _i, _i, _i, _i, _i, _i]),
    "sht_plan_s2_opts": (_i, [C.POINTER(_vp), _i, _i, _i, _i, _i, _i, _i, C.c_uint]),
    "sht_plan_batch": (_i, [_vp]),
    "sht_plan_workspace_bytes": (_sz, [_vp]),
    "sht_plan_set_workspace": (_i, [_vp, _vp, _sz, _vp]),
    "sht_plan_destroy": (_i, [_vp]),
    "s2_forward_plan": (_i, [_vp, _vp, _vp, _vp]),
    "s2_inverse_plan": (_i, [_vp, _vp, _vp, _vp]),
    "s2_forward_iter_plan": (_i, [_vp, _vp, _vp, _i, _vp]),
    "so3_forward_plan": (_i, [_vp, _vp, _vp, _vp]),
    "so3_inverse_plan": (_i, [_vp, _vp, _vp, _vp]),
    "s2_forward_adjoint_plan": (_i, [_vp, _vp, _vp, _vp]),
    "s2_inverse_adjoint_plan": (_i, [_vp, _vp, _vp, _vp]),
    "s2_theta_forward_adjoint_plan": (_i, [_vp, _vp, _vp, _vp]),
    "s2_theta_inverse_adjoint_plan": (_i, [_vp, _vp, _vp, _vp]),
    "sht_plan_set_shard": (_i, [_vp, _i, _i]),
    "sht_plan_shard_range": (_i, [_vp, _i, C.POINTER(_i), C.POINTER(_i)]),
    "sht_plan_ntheta": (_i, [_vp, _i]),
    "s2_theta_inverse_plan": (_i, [_vp, _vp, _vp, _vp]),
    "s2_theta_forward_plan": (_i, [_vp, _vp, _vp, _vp]),
    "sht_plan_enable_timing": (_i, [_vp, _i]),
    "sht_plan_timings": (_i, [_vp, C.POINTER(C.c_float)]),
    "sht_plan_stage_bytes": (_i, [_vp, C.POINTER(C.c_double)]),
    "s2_forward": (_i, [_i, _i, _i, _i, _vp, _vp, _vp]),
    "s2_inverse": (_i, [_i, _i, _i, _i, _vp, _vp, _vp]),
    "so3_forward": (_i, [_i, _i, _vp, _vp, _vp]),
    "so3_inverse": (_i, [_i, _i, _vp, _vp, _vp]),
    "sht_cache_clear": (_i, []),
    "s2_forward_host": (_i, [_i, _i, _i, _i, _vp, _vp, _vp]),
    "s2_inverse_host": (_i, [_i, _i, _i, _i, _vp, _vp, _vp]),
    "so3_forward_host": (_i, [_i, _i, _vp, _vp, _vp]),
    "so3_inverse_host": (_i, [_i, _i, _vp, _vp, _vp]),
    "sht_peak": (_i, [_i, _i, C.POINTER(C.c_double), C.POINTER(C.c_float), _vp]),
    "sht_fp64_peak": (_i, [_i, C.POINTER(C.c_double), C.POINTER(C.c_float), _vp]),
    "sht_launch_count": (C.c_long, [_i]),
    "sht_plan_dsteps": (C.c_double, [_vp, _i]),
    "sht_plan_flops": (C.c_double, [_vp, _i]),
    "sht_plan_skip_fraction": (C.c_double, [_vp, _i]),
    "sht_version": (C.c_char_p, []),
    "s2_theta_inverse_noalloc": (_i, [_i, _i, _i, C.POINTER(C.c_double), _vp, _vp, _vp, C.c_char_p, _sz]),
}

_lib = None


def lib():
    """Load the CUDA library (once).  Raises if it has not been built -- there is no CPU path."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2311_14670_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


class ShtError(RuntimeError):
    pass


def check(status):
    if status != 0:
        L = lib()
        raise ShtError(f"{L.sht_status_string(status).decode()} [{L.sht_last_error().decode()}]")
