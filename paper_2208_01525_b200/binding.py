"""Thin ctypes binding of libu1u1.so (include/u1u1.h): same names, argument marshalling only.

Every step of the path runs in the CUDA kernels of the library; there is no CPU or PyTorch fallback:
if the shared library is missing, `load()` raises.  PyTorch is used by the `Lattice` helper only to
own device memory and the stream.
"""
from __future__ import annotations

import ctypes
import os

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libu1u1.so")

DIAG_LEN = 48
GAUSS_LEN = 8
STATIC_MAX_N = 1024        # U1U1_STATIC_MAX_N
SEG_LEN = 8
SEG_SLOTS = ["N_pq", "L_pq", "l_pq", "cells_kept", "segments_all", "cells_all", "largest", "cells_mask"]
DIAG_SLOTS = ["tau", "a", "c", "sumW_p", "sumW_q", "cells_p", "cells_q", "cells_pq", "near_p", "near_q",
              "maxW", "sum_L", "sum_kin_L", "sum_grad_L", "sum_kin_V", "sum_grad_V", "sum_vint", "sum_kin",
              "sum_grad", "sum_elec", "sum_mag", "sum_pot", "L_p", "L_q", "L_pq", "xi_p", "xi_q", "xi_pq",
              "xi_W", "xi_L", "f_total", "f_p", "v2_L", "v2_pq", "energy", "cells_pq_tol_p", "cells_pq_tol_q", "L_pq_tol",
              "max_theta", "gauss_l2_p", "gauss_rho_p", "gauss_max_p", "gauss_rel_p", "gauss_l2_q", "gauss_rho_q",
              "gauss_max_q", "gauss_rel_q", "v2_valid"]
ERRORS = {-1: "EINVAL", -2: "ESIZE", -3: "EPARAM", -4: "ESTATE", -5: "ECUDA", -6: "EUNSTABLE"}


class Params(ctypes.Structure):
    """u1u1_params (include/u1u1.h).  Defaults: the paper's validation couplings."""
    _fields_ = [("struct_size", ctypes.c_uint32), ("init_kind", ctypes.c_int32),
                ("lambda1", ctypes.c_double), ("lambda2", ctypes.c_double),
                ("e1", ctypes.c_double), ("e2", ctypes.c_double),
                ("eta1", ctypes.c_double), ("eta2", ctypes.c_double),
                ("kappa", ctypes.c_double), ("dtau", ctypes.c_double),
                ("tau_norm", ctypes.c_double), ("friction", ctypes.c_double),
                ("smooth_width", ctypes.c_double), ("smooth_trunc", ctypes.c_int32),
                ("kernel_variant", ctypes.c_int32), ("range_reduce", ctypes.c_int32), ("reserved", ctypes.c_int32)]

    def __init__(self, **kw):
        """kernel_variant = 0..7 (include/u1u1.h).  For the tests' convenience a value of variant + 16 * switches is split
        here: the switches (include/u1u1_tuning.h) go to `self.tuning`, which Lattice hands to u1u1_set_tuning, and the old
        switch 2048 becomes the named field range_reduce = 1.  The C struct never sees more than 0..7."""
        d = dict(init_kind=0, lambda1=2.0, lambda2=2.0, e1=1.0, e2=1.0, eta1=1.0, eta2=1.0, kappa=0.9,
                 dtau=0.1, tau_norm=1.0, friction=1.0, smooth_width=5.0, smooth_trunc=20, kernel_variant=0,
                 range_reduce=0, reserved=0)
        d.update(kw)
        kv = int(d["kernel_variant"])
        self.tuning = (kv >> 4) & 2047
        if (kv >> 4) & 2048:
            d["range_reduce"] = 1
        d["kernel_variant"] = kv & 15
        super().__init__(struct_size=ctypes.sizeof(Params), **d)


class U1U1Error(RuntimeError):
    pass


_lib = None
SYMBOLS = ["u1u1_state_bytes", "u1u1_scratch_bytes", "u1u1_aux_bytes", "u1u1_set_aux", "u1u1_create", "u1u1_destroy", "u1u1_last_error",
           "u1u1_configure", "u1u1_init_fields", "u1u1_set_params", "u1u1_set_time", "u1u1_step", "u1u1_cool",
           "u1u1_diagnostics", "u1u1_gauss_violation", "u1u1_gauss_violation_static", "u1u1_export_state", "u1u1_import_state",
           "u1u1_export_state_host", "u1u1_import_state_host", "u1u1_export_windings", "u1u1_export_block", "u1u1_launch_count", "u1u1_pq_segments", "u1u1_export_labels", "u1u1_import_state_tiled",
           "u1u1_slab_state_bytes", "u1u1_configure_slab", "u1u1_set_slab_peers", "u1u1_init_slab", "u1u1_export_slab",
           "u1u1_import_slab", "u1u1_push_halos", "u1u1_slab_scratch_bytes", "u1u1_push_diag_halos",
           "u1u1_slab_diagnostics_partial", "u1u1_slab_diagnostics_finish"]
TUNING_SYMBOLS = ["u1u1_set_tuning"]          # include/u1u1_tuning.h: experimental switches, outside the supported boundary
SLAB_NRAW, SLAB_NSUM = 28, 24


def load():
    """dlopen libu1u1.so (built in-tree by paper_2208_01525_b200.build).  Fails loudly if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise U1U1Error(f"{LIB_PATH} not found: run `python -m paper_2208_01525_b200.build` "
                        "(there is no CPU fallback)")
    L = ctypes.CDLL(LIB_PATH)
    vp, d, i32, u64 = ctypes.c_void_p, ctypes.c_double, ctypes.c_int32, ctypes.c_uint64
    dp, pp = ctypes.POINTER(ctypes.c_double), ctypes.POINTER(Params)
    L.u1u1_state_bytes.argtypes = [i32]; L.u1u1_state_bytes.restype = ctypes.c_size_t
    L.u1u1_scratch_bytes.argtypes = [i32]; L.u1u1_scratch_bytes.restype = ctypes.c_size_t
    L.u1u1_aux_bytes.argtypes = [i32]; L.u1u1_aux_bytes.restype = ctypes.c_size_t
    L.u1u1_set_aux.argtypes = [vp, vp, ctypes.c_size_t]
    L.u1u1_create.argtypes = [ctypes.POINTER(vp), vp, ctypes.c_size_t, vp, ctypes.c_size_t, vp]
    L.u1u1_destroy.argtypes = [vp]; L.u1u1_destroy.restype = None
    L.u1u1_last_error.argtypes = [vp]; L.u1u1_last_error.restype = ctypes.c_char_p
    L.u1u1_configure.argtypes = [vp, i32, d, pp]
    L.u1u1_init_fields.argtypes = [vp, u64, i32, d, pp]
    L.u1u1_set_params.argtypes = [vp, pp]
    L.u1u1_set_tuning.argtypes = [vp, ctypes.c_uint32]
    L.u1u1_set_time.argtypes = [vp, d, d, d]
    L.u1u1_step.argtypes = [vp, i32, d, d, d]
    L.u1u1_cool.argtypes = [vp, i32, d]
    L.u1u1_diagnostics.argtypes = [vp, dp]
    L.u1u1_gauss_violation.argtypes = [vp, dp]
    L.u1u1_gauss_violation_static.argtypes = [vp, i32, d, d, d, d, vp, vp, ctypes.c_char_p, ctypes.c_size_t]
    L.u1u1_export_state.argtypes = [vp, vp]
    L.u1u1_import_state.argtypes = [vp, vp]
    L.u1u1_export_state_host.argtypes = [vp, vp]
    L.u1u1_import_state_host.argtypes = [vp, vp]
    L.u1u1_export_windings.argtypes = [vp, i32, vp, vp, vp]
    L.u1u1_export_block.argtypes = [vp, i32, i32, i32, i32, i32, i32, vp]
    L.u1u1_pq_segments.argtypes = [vp, i32, i32, dp]
    L.u1u1_export_labels.argtypes = [vp, vp]
    L.u1u1_import_state_tiled.argtypes = [vp, vp, i32]
    L.u1u1_launch_count.argtypes = [vp]; L.u1u1_launch_count.restype = u64
    L.u1u1_slab_state_bytes.argtypes = [i32, i32]; L.u1u1_slab_state_bytes.restype = ctypes.c_size_t
    L.u1u1_configure_slab.argtypes = [vp, i32, i32, ctypes.c_int64, d, pp]
    L.u1u1_set_slab_peers.argtypes = [vp, vp, vp]
    L.u1u1_init_slab.argtypes = [vp, u64]
    L.u1u1_export_slab.argtypes = [vp, vp]
    L.u1u1_import_slab.argtypes = [vp, vp]
    L.u1u1_push_halos.argtypes = [vp]
    L.u1u1_slab_scratch_bytes.argtypes = [i32, i32]; L.u1u1_slab_scratch_bytes.restype = ctypes.c_size_t
    L.u1u1_push_diag_halos.argtypes = [vp]
    L.u1u1_slab_diagnostics_partial.argtypes = [vp, dp]
    L.u1u1_slab_diagnostics_finish.argtypes = [vp, dp, ctypes.c_int64, dp]
    _lib = L
    return L


def state_bytes(N: int) -> int:
    return load().u1u1_state_bytes(N)


def scratch_bytes(N: int) -> int:
    return load().u1u1_scratch_bytes(N)
