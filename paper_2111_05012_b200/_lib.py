"""ctypes loader for liblqcd_b200.so (the C ABI of include/lqcd_b200.h).

There is no CPU fallback: if the library is missing and cannot be built with nvcc, loading raises.
"""
from __future__ import annotations

import ctypes as C
import os

from . import build as _build

_lib = None

c_int4 = C.c_int * 4
_vp, _ci, _cu, _cf, _cd = C.c_void_p, C.c_int, C.c_uint, C.c_float, C.c_double
_i4 = C.POINTER(C.c_int)
_i8 = C.POINTER(C.c_int)       # int[8]
_p8 = C.POINTER(C.c_void_p)    # void*[8]: host array of device pointers
APPLY_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p)             # lqcd_apply_fn
REDUCE_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_size_t, C.c_int, C.c_void_p, C.c_void_p)   # lqcd_reduce_fn

# name -> (restype, argtypes); every symbol include/lqcd_b200.h declares
SIGNATURES = {
    "lqcd_version": (_ci, []),
    "lqcd_last_error": (C.c_char_p, []),
    "lqcd_launch_count": (C.c_ulonglong, []),
    "lqcd_set_fine_tile": (_ci, [_i4]),
    "lqcd_set_knob": (_ci, [C.c_char_p, _ci]),
    "lqcd_native_spinor_reals": (C.c_size_t, [_i4]),
    "lqcd_native_gauge_reals": (C.c_size_t, [_i4, _cu]),
    "lqcd_native_clover_reals": (C.c_size_t, [_i4]),
    "lqcd_native_nullvecs_reals": (C.c_size_t, [_i4, _i4, _ci]),
    "lqcd_native_coarse_vec_reals": (C.c_size_t, [_i4, _ci]),
    "lqcd_native_coarse_mat_reals": (C.c_size_t, [_i4, _ci]),
    "lqcd_coarse_mult_half_noalloc_f32": (_ci, [_vp, _vp, _vp, _i4, _ci, _cu, _vp]),
    "lqcd_native_coarse_half_reals": (C.c_size_t, [_i4, _ci]),
    "lqcd_coarse_half_workspace_bytes": (C.c_size_t, [_i4, _ci, _ci]),
    "lqcd_host_workspace_bytes": (C.c_size_t, [_i4, _i4, _ci]),
    "lqcd_host_workspace_bytes_f64": (C.c_size_t, [_i4, _i4, _ci]),
    "lqcd_galerkin_workspace_bytes": (C.c_size_t, [_i4, _i4, _ci, _ci]),
    "lqcd_orthonormalize_degenerate_count": (C.c_longlong, [_vp]),
    "lqcd_mr_workspace_bytes": (C.c_size_t, [_i4, _i4, _ci]),
    "lqcd_coarse_bicgstab_workspace_bytes": (C.c_size_t, [_i4, _ci, _ci]),
    "lqcd_mg_workspace_bytes": (C.c_size_t, [_i4, _i4, _ci, _ci]),
    "lqcd_mg_mrhs_workspace_bytes": (C.c_size_t, [_i4, _i4, _ci, _ci, _ci]),
    "lqcd_coarse_bicgstab_mrhs_workspace_bytes": (C.c_size_t, [_i4, _ci, _ci, _ci]),
    "lqcd_halo_face_reals": (C.c_size_t, [_i4, _ci]),
    "lqcd_coarse_halo_face_reals": (C.c_size_t, [_i4, _ci, _ci]),
}
for _p, _k in (("f32", _cf), ("f64", _cd)):
    SIGNATURES.update({
        f"lqcd_pack_spinor_{_p}": (_ci, [_vp, _vp, _i4, _vp]),
        f"lqcd_unpack_spinor_{_p}": (_ci, [_vp, _vp, _i4, _vp]),
        f"lqcd_pack_gauge_{_p}": (_ci, [_vp, _vp, _i4, _cu, _vp]),
        f"lqcd_pack_clover_{_p}": (_ci, [_vp, _vp, _i4, _vp]),
        f"lqcd_unpack_clover_{_p}": (_ci, [_vp, _vp, _i4, _vp]),
        f"lqcd_clover_from_links_{_p}": (_ci, [_vp, _vp, _k, _k, _i4, _vp]),
        f"lqcd_orthonormalize_blocks_{_p}": (_ci, [_vp, _i4, _i4, _ci, _vp]),
        f"lqcd_galerkin_coarse_{_p}": (_ci, [_vp, _vp, _vp, _vp, _k, _i4, _i4, _i4, _ci, _vp, _vp]),
        f"lqcd_pack_nullvec_{_p}": (_ci, [_vp, _vp, _ci, _i4, _i4, _ci, _vp]),
        f"lqcd_pack_coarse_half_{_p}": (_ci, [_vp, _vp, _i4, _ci, _vp]),
        f"lqcd_coarse_mult_half_{_p}": (_ci, [_vp, _vp, _vp, _i4, _ci, _cu, _vp, _vp]),
        f"lqcd_unpack_nullvec_{_p}": (_ci, [_vp, _vp, _ci, _i4, _i4, _ci, _vp]),
        f"lqcd_wilson_clover_mult_{_p}": (_ci, [_vp, _vp, _vp, _vp, _k, _i4, _i4, _cu, _vp]),
        f"lqcd_wilson_clover_dd_mult_{_p}": (_ci, [_vp, _vp, _vp, _vp, _k, _i4, _i4, _i4, _cu, _vp]),
        f"lqcd_coarse_mult_{_p}": (_ci, [_vp, _vp, _vp, _i4, _ci, _cu, _vp]),
        f"lqcd_restrict_{_p}": (_ci, [_vp, _vp, _vp, _i4, _i4, _ci, _vp]),
        f"lqcd_prolong_{_p}": (_ci, [_vp, _vp, _vp, _i4, _i4, _ci, _vp]),
        f"lqcd_wilson_clover_residual_{_p}": (_ci, [_vp, _vp, _vp, _vp, _vp, _k, _i4, _i4, _cu, _vp]),
        f"lqcd_block_dotc_{_p}": (_ci, [_vp, _vp, _vp, _i4, _i4, _vp]),
        f"lqcd_block_caxpy_{_p}": (_ci, [_vp, _vp, _vp, _i4, _i4, _vp]),
        f"lqcd_mr_domain_solve_{_p}": (_ci, [_vp, _vp, _vp, _vp, _k, _i4, _i4, _i4, _cu, _ci, _vp, _vp]),
        f"lqcd_coarse_bicgstab_{_p}": (_ci, [_vp, _vp, _vp, _vp, _i4, _ci, _ci, _vp, _vp]),
        f"lqcd_coarse_bicgstab_half_{_p}": (_ci, [_vp, _vp, _vp, _vp, _i4, _ci, _ci, _vp, _vp]),
        f"lqcd_mg_vcycle_{_p}": (_ci, [_vp, _vp, _vp, _vp, _k, _i4, _i4, _i4, _ci, _vp, _vp, _ci, _ci, _ci, _vp, _vp]),
        f"lqcd_mg_vcycle_half_{_p}": (_ci, [_vp, _vp, _vp, _vp, _k, _i4, _i4, _i4, _ci, _vp, _vp, _ci, _ci, _ci, _vp, _vp]),
        f"lqcd_coarse_mult_mrhs_{_p}": (_ci, [_vp, _vp, _vp, _i4, _ci, _ci, _cu, _vp]),
        f"lqcd_wilson_clover_mult_mrhs_{_p}": (_ci, [_vp, _vp, _vp, _vp, _k, _i4, _i4, _ci, _cu, _vp]),
        f"lqcd_restrict_mrhs_{_p}": (_ci, [_vp, _vp, _vp, _i4, _i4, _ci, _ci, _vp]),
        f"lqcd_coarse_bicgstab_mrhs_{_p}": (_ci, [_vp, _vp, _vp, _vp, _i4, _ci, _ci, _ci, _vp, _vp]),
        f"lqcd_prolong_mrhs_{_p}": (_ci, [_vp, _vp, _vp, _i4, _i4, _ci, _ci, _vp]),
        f"lqcd_mg_vcycle_mrhs_{_p}": (_ci, [_vp, _vp, _vp, _vp, _k, _i4, _i4, _i4, _ci, _vp, _vp, _ci, _ci, _ci, _ci, _vp,
                                           _vp]),
        f"lqcd_sap_mrhs_{_p}": (_ci, [_vp, _vp, _vp, _vp, _vp, _k, _i4, _i4, _i4, _ci, _ci, _ci, _cu, _vp, _vp]),
        f"lqcd_sap_{_p}": (_ci, [_vp, _vp, _vp, _vp, _vp, _k, _i4, _i4, _i4, _ci, _ci, _cu, _vp, _vp]),
        f"lqcd_coarse_bicgstab_hooks_{_p}": (_ci, [_vp, _vp, _vp, _i4, _ci, _ci, APPLY_FN, REDUCE_FN, _vp, _vp, _vp]),
        f"lqcd_coarse_halo_pack_{_p}": (_ci, [_p8, _vp, _i4, _ci, _cu, _vp]),
        f"lqcd_coarse_mult_interior_{_p}": (_ci, [_vp, _vp, _vp, _i4, _ci, _cu, _cu, _vp]),
        f"lqcd_coarse_halo_add_{_p}": (_ci, [_vp, _p8, _vp, _i4, _ci, _cu, _cu, _vp]),
        f"lqcd_wilson_clover_halo_pack_{_p}": (_ci, [_p8, _vp, _vp, _i4, _cu, _cu, _vp]),
        f"lqcd_wilson_clover_mult_interior_{_p}": (_ci, [_vp, _vp, _vp, _vp, _k, _i4, _i4, _cu, _cu, _vp]),
        f"lqcd_wilson_clover_residual_interior_{_p}": (_ci, [_vp, _vp, _vp, _vp, _vp, _k, _i4, _i4, _i4, _cu, _cu,
                                                             _vp]),
        f"lqcd_wilson_clover_halo_add_{_p}": (_ci, [_vp, _p8, _vp, _k, _i4, _i8, _cu, _cu, _vp]),
    })
for _p, _k in (("f32", _cf), ("f64", _cd)):
    SIGNATURES.update({
        f"lqcd_wilson_clover_mult_host_{_p}": (_ci, [_vp, _vp, _vp, _vp, _k, _i4, _i4, _cu, _vp, _vp]),
        f"lqcd_coarse_mult_host_{_p}": (_ci, [_vp, _vp, _vp, _i4, _ci, _cu, _vp, _vp]),
        f"lqcd_restrict_host_{_p}": (_ci, [_vp, _vp, _vp, _i4, _i4, _ci, _vp, _vp]),
        f"lqcd_prolong_host_{_p}": (_ci, [_vp, _vp, _vp, _i4, _i4, _ci, _vp, _vp]),
    })


def lib_path() -> str:
    return _build.LIB


def load():
    """Load (building first if the sources are newer and nvcc is present) and type every entry point."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if _build.stale():
        try:
            _build.build()
        except Exception as e:  # no nvcc on this box
            if not os.path.exists(path):
                raise RuntimeError(
                    f"liblqcd_b200.so is missing and could not be built ({e}); there is no CPU fallback") from e
            if os.environ.get("LQCD_REQUIRE_FRESH"):
                raise RuntimeError(f"liblqcd_b200.so is older than its sources and the rebuild failed ({e})") from e
            import warnings
            warnings.warn(f"liblqcd_b200.so is OLDER than its sources and the rebuild failed ({e}): loading the stale "
                          "library (set LQCD_REQUIRE_FRESH=1 to make this an error)", RuntimeWarning, stacklevel=2)
    lib = C.CDLL(path)
    for name, (res, args) in SIGNATURES.items():
        fn = getattr(lib, name)  # AttributeError if the header and the library disagree
        fn.restype = res
        fn.argtypes = args
    _lib = lib
    return lib
