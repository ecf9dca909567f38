"""ctypes loader for the C-ABI library (include/cclr.h).  No arithmetic here: argument marshalling only.

The product path fails loudly when the CUDA library is missing: there is no CPU fallback.
"""
import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libcclr.so")

c128_p = C.c_void_p  # device or host pointer to interleaved complex128


class EriPacked(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in ("oooo", "ooov", "oovv", "ovvo", "ovvv", "vvvv")]


class SolveInfo(C.Structure):
    _fields_ = [("iterations", C.c_int), ("sigma_calls", C.c_int), ("subspace", C.c_int), ("converged", C.c_int),
                ("max_residual", C.c_double), ("seconds", C.c_double)]


class CcsdInfo(C.Structure):
    _fields_ = [("iterations", C.c_int), ("converged", C.c_int), ("sigma_calls", C.c_int), ("residual", C.c_double),
                ("energy_re", C.c_double), ("energy_im", C.c_double), ("seconds", C.c_double)]


class EomInfo(C.Structure):
    _fields_ = [("iterations", C.c_int), ("sigma_calls", C.c_int), ("subspace", C.c_int), ("converged", C.c_int),
                ("max_residual", C.c_double), ("seconds", C.c_double)]


class Complex(C.Structure):
    _fields_ = [("re", C.c_double), ("im", C.c_double)]


# name -> (restype, argtypes); must list every symbol include/cclr.h declares (tests/test_abi.py checks this)
SIGNATURES = {
    "cclr_create": (C.c_int, [C.c_int, C.c_int, c128_p, C.POINTER(EriPacked), c128_p, c128_p, C.c_uint, C.c_void_p,
                              C.POINTER(C.c_void_p)]),
    "cclr_sigma": (C.c_int, [C.c_void_p, c128_p, c128_p, C.c_int, C.c_double, C.c_double, c128_p, c128_p]),
    "cclr_sigma_left": (C.c_int, [C.c_void_p, c128_p, c128_p, C.c_int, C.c_double, C.c_double, c128_p, c128_p]),
    "cclr_solve": (C.c_int, [C.c_void_p, c128_p, c128_p, C.c_int, C.POINTER(C.c_double), C.c_int, C.c_double,
                             C.c_double, C.c_int, c128_p, c128_p, C.POINTER(SolveInfo)]),
    "cclr_solve_left": (C.c_int, [C.c_void_p, c128_p, c128_p, C.c_int, C.POINTER(C.c_double), C.c_int, C.c_double,
                                  C.c_double, C.c_int, c128_p, c128_p, C.POINTER(SolveInfo)]),
    "cclr_lambda": (C.c_int, [C.c_void_p, C.c_double, C.c_int, c128_p, c128_p, C.POINTER(SolveInfo)]),
    "cclr_eta": (C.c_int, [C.c_void_p, c128_p, c128_p, c128_p, C.c_int, c128_p, c128_p]),
    "cclr_response_ci": (C.c_int, [C.c_void_p, c128_p, c128_p, C.c_double, C.c_double, C.c_double, C.c_int,
                                   C.POINTER(Complex), C.POINTER(SolveInfo)]),
    "cclr_response_ci_tensor": (C.c_int, [C.c_void_p, c128_p, C.c_int, C.POINTER(C.c_double), C.c_int, C.c_double, C.c_double,
                                          C.c_int, C.POINTER(Complex), C.POINTER(SolveInfo)]),
    "cclr_xfy": (C.c_int, [C.c_int, C.c_int, c128_p, C.POINTER(EriPacked), c128_p, c128_p, c128_p, c128_p, c128_p, c128_p,
                           c128_p, c128_p, C.c_void_p, C.POINTER(Complex)]),
    "cclr_response_cc": (C.c_int, [C.c_void_p, C.POINTER(EriPacked), c128_p, c128_p, C.c_double,
                                   C.c_double, C.c_double, C.c_int, C.POINTER(Complex), C.POINTER(SolveInfo)]),
    "cclr_f_transform": (C.c_int, [C.c_void_p, C.POINTER(EriPacked), c128_p, c128_p, c128_p, c128_p, C.c_int, c128_p, c128_p]),
    "cclr_xi": (C.c_int, [C.c_void_p, c128_p, c128_p, c128_p]),
    "cclr_property": (C.c_int, [C.c_void_p, c128_p, c128_p, c128_p, c128_p, C.c_int, C.POINTER(Complex)]),
    "cclr_ccsd": (C.c_int, [C.c_int, C.c_int, c128_p, C.POINTER(EriPacked), c128_p, c128_p, C.c_double, C.c_int, C.c_void_p,
                            C.POINTER(CcsdInfo)]),
    "cclr_eom": (C.c_int, [C.c_void_p, C.c_int, C.c_double, C.c_int, C.c_void_p, c128_p, c128_p, C.POINTER(EomInfo)]),
    "cclr_host_eigen": (C.c_int, [C.c_int, c128_p, c128_p, c128_p]),
    "cclr_ccsd_residual": (C.c_int, [C.c_int, C.c_int, c128_p, C.POINTER(EriPacked), c128_p, c128_p, C.c_int, C.c_void_p,
                                     c128_p, c128_p]),
    "cclr_set_max_subspace": (C.c_int, [C.c_void_p, C.c_int]),
    "cclr_destroy": (None, [C.c_void_p]),
    "cclr_strerror": (C.c_char_p, [C.c_int]),
    "cclr_last_cuda_error": (C.c_int, []),
    "cclr_last_error_message": (C.c_char_p, []),
    "cclr_sigma_host": (C.c_int, [C.c_void_p, c128_p, c128_p, C.c_int, C.c_double, C.c_double, c128_p, c128_p]),
    "cclr_zgemm": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_int, C.POINTER(Complex), c128_p, C.c_long, C.c_int,
                             c128_p, C.c_long, C.c_int, C.c_int, C.POINTER(Complex), c128_p, C.c_long, C.c_int,
                             C.c_long, C.c_long, C.c_long, C.c_int]),
    "cclr_property_noalloc": (C.c_int, [C.c_void_p, c128_p, c128_p, c128_p, c128_p, C.c_long, C.c_long, C.c_int, c128_p]),
    "cclr_set_gemm_path": (C.c_int, [C.c_void_p, C.c_int]),
    "cclr_gemm_slices": (C.c_int, [C.c_void_p]),
    "cclr_zgemm_oz": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_int, C.POINTER(Complex), c128_p, C.c_long, C.c_int,
                                c128_p, C.c_long, C.c_int, C.c_int, C.POINTER(Complex), c128_p, C.c_long, C.c_int, C.c_int,
                                C.c_int, C.POINTER(C.c_double)]),
    "cclr_vec_block_lincomb": (C.c_int, [C.c_void_p, C.c_int, c128_p, C.c_long, c128_p, C.c_long, c128_p, c128_p, C.c_long, C.c_int,
                                         C.c_long, C.c_void_p, c128_p, c128_p, C.c_long]),
    "cclr_vec_dots": (C.c_int, [C.c_void_p, c128_p, C.c_int, c128_p, C.c_int, C.c_long, C.c_long, C.POINTER(Complex)]),
    "cclr_host_shifted_solve": (C.c_int, [C.c_int, c128_p, c128_p, C.c_int, c128_p, c128_p]),
    "cclr_ladder": (C.c_int, [C.c_void_p, c128_p, C.c_int, c128_p]),
    "cclr_ring": (C.c_int, [C.c_void_p, c128_p, c128_p]),
    "cclr_get_intermediate": (C.c_long, [C.c_void_p, C.c_char_p, c128_p, C.c_long]),
    "cclr_get_intermediate_slice": (C.c_long, [C.c_void_p, C.c_char_p, C.c_long, C.c_long, c128_p]),
    "cclr_kernel_launches": (C.c_ulonglong, []),
    "cclr_ctx_bytes": (C.c_size_t, [C.c_void_p]),
    "cclr_set_profiling": (C.c_int, [C.c_void_p, C.c_int]),
    "cclr_last_sigma_ms": (C.c_int, [C.c_void_p, C.POINTER(C.c_double)]),
    "cclr_sigma_op_count": (C.c_int, [C.c_void_p]),
    "cclr_sigma_op_text": (C.c_char_p, [C.c_void_p, C.c_int]),
    "cclr_last_sigma_op_ms": (C.c_int, [C.c_void_p, C.POINTER(C.c_double), C.c_int]),
    "cclr_fp64_tensor_peak": (C.c_int, [C.c_void_p, C.c_int, C.POINTER(C.c_double)]),
    "cclr_fp64_pipe_probe": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.POINTER(C.c_double)]),
    "cclr_hbm_copy_peak": (C.c_int, [C.c_void_p, C.c_size_t, C.POINTER(C.c_double)]),
}

_lib = None


def load():
    """Load libcclr.so (built by ``python -m paper_2307_14296_b200.build``) and set the prototypes."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("libcclr.so is missing: run `python -m paper_2307_14296_b200.build` (there is no "
                               "CPU fallback)")
        lib = C.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(lib, name)  # AttributeError if the library does not export a declared symbol
            fn.restype, fn.argtypes = res, args
        _lib = lib
    return _lib


class CclrError(RuntimeError):
    def __init__(self, code, where):
        lib = load()
        msg = lib.cclr_strerror(code).decode()
        extra = " (cuda error %d)" % lib.cclr_last_cuda_error() if code == -3 else ""
        detail = lib.cclr_last_error_message().decode()
        if detail:
            extra += ": " + detail
        super().__init__("%s: %s%s" % (where, msg, extra))
        self.code = code


def check(code, where):
    if code != 0:
        raise CclrError(code, where)
