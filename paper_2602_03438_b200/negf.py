"""Thin ctypes binding of include/negf.h - same names, argument marshalling only.

Every step of the path runs in the CUDA kernels of libnegf_b200.so; this module only turns
torch tensors (device memory + streams: plumbing) into pointers.  There is NO CPU fallback:
importing this module raises if the library is missing, and `Context()` raises without a
compute-capability-10.x GPU.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libnegf_b200.so")
if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2602_03438_b200.build` "
                      "(or __graft_entry__.build()); there is no CPU fallback")
lib = C.CDLL(LIB_PATH)

PROF_GEMM, PROF_INVERSE, PROF_ELEMENTWISE, PROF_OBSERVABLES, PROF_FUSED = range(5)
PROF_NAMES = ("gemm", "inverse", "elementwise", "observables", "fused")
OK, EINVAL, ENOWORKSPACE, EUNSUPPORTED, ECUDA, ENOSTATE, ESTATICLIMIT = 0, -1, -2, -3, -4, -5, -6
STATIC_SCRATCH_BYTES = 16 << 20
SIGMA_NONE, SIGMA_SCALAR, SIGMA_BT = 0, 1, 2
KEEP_SWEEP = 1
OPT_GRAPH_LOOPS = 1
OPT_GEMM_3M = 2
OPT_INV_TENSOR = 3
OPT_ENERGY_GROUPS = 4
OPT_INV_PANEL = 5
OPT_INV_LOOKAHEAD = 6
OPT_INV_OUTER = 7
OPT_FUSED_SMALL = 8
OPT_PDL = 9


class c128(C.Structure):
    _fields_ = [("re", C.c_double), ("im", C.c_double)]


class Problem(C.Structure):
    _fields_ = [("n_blocks", C.c_int), ("block_size", C.c_int), ("n_energy", C.c_int),
                ("H_diag", C.c_void_p), ("H_upper", C.c_void_p), ("S_diag", C.c_void_p),
                ("S_upper", C.c_void_p), ("energy", C.c_void_p), ("eta", C.c_double),
                ("n_k", C.c_int), ("k_index", C.c_void_p)]


class Sigma(C.Structure):
    _fields_ = [("kind", C.c_int), ("scalar", C.c_void_p), ("diag", C.c_void_p), ("upper", C.c_void_p),
                ("lower", C.c_void_p), ("left", C.c_void_p), ("right", C.c_void_p)]


class Lead(C.Structure):
    _fields_ = [("H_d", C.c_void_p), ("H_u", C.c_void_p), ("S_d", C.c_void_p), ("S_u", C.c_void_p)]


class ObcOut(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in
                ("sigma_r", "gamma", "sigma_lesser", "sigma_greater", "g_surface", "fermi", "iters", "status")]


class HostOutputs(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in
                ("GR_diag", "GR_upper", "GR_lower", "GL_diag", "GL_upper", "GG_diag", "GG_upper",
                 "density", "ldos", "transmission", "bond_current", "contact_current", "info")]


class DeviceOutputs(C.Structure):
    _fields_ = [("left", ObcOut), ("right", ObcOut)] + [(k, C.c_void_p) for k in
                ("GR_diag", "GR_upper", "GR_lower", "GR_corner", "GL_diag", "GL_upper", "GG_diag", "GG_upper",
                 "density", "ldos", "transmission", "bond_current", "contact_current", "info_r", "info_x")]


EXPORTS = ["negf_create", "negf_destroy", "negf_set_stream", "negf_workspace_bytes", "negf_set_workspace",
           "negf_set_option", "negf_strerror", "negf_last_cuda_error", "negf_launch_count", "negf_obc_graph_kernels",
           "negf_profile_enable", "negf_profile_read", "negf_obc_decimate", "negf_obc_decimate_pair",
           "negf_rgf_retarded", "negf_rgf_lesser_greater", "negf_observables", "negf_energy_convolve", "negf_pipeline_device",
           "negf_pipeline_host_bytes",
           "negf_pipeline_host", "negf_zgemm_batched", "negf_zinverse_batched", "negf_zinverse_batched_static",
           "negf_fp64_peak"]

_P = C.c_void_p
lib.negf_create.argtypes = [C.POINTER(_P), C.c_int]
lib.negf_destroy.argtypes = [_P]
lib.negf_set_stream.argtypes = [_P, _P]
lib.negf_workspace_bytes.argtypes = [C.POINTER(Problem), C.c_int, C.c_int, C.POINTER(C.c_size_t)]
lib.negf_set_workspace.argtypes = [_P, _P, C.c_size_t]
lib.negf_set_option.argtypes = [_P, C.c_int, C.c_int]
lib.negf_strerror.argtypes = [C.c_int]
lib.negf_strerror.restype = C.c_char_p
lib.negf_last_cuda_error.argtypes = [_P]
lib.negf_launch_count.argtypes = [_P]
lib.negf_launch_count.restype = C.c_longlong
lib.negf_obc_graph_kernels.argtypes = [_P]
lib.negf_obc_graph_kernels.restype = C.c_longlong
lib.negf_profile_enable.argtypes = [_P, C.c_int]
lib.negf_profile_read.argtypes = [_P, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_longlong), C.c_int]
lib.negf_obc_decimate.argtypes = [_P, C.POINTER(Problem), C.POINTER(Lead), C.c_int, C.c_double, C.c_double,
                                  C.c_double, C.c_int, _P, _P, _P, _P, _P, _P, _P, _P]
lib.negf_obc_decimate_pair.argtypes = [_P, C.POINTER(Problem), C.POINTER(Lead), C.POINTER(Lead), C.c_double,
                                       C.c_double, C.c_double, C.c_double, C.c_int, C.POINTER(ObcOut),
                                       C.POINTER(ObcOut)]
lib.negf_rgf_retarded.argtypes = [_P, C.POINTER(Problem), C.POINTER(Sigma), _P, _P, _P, _P, C.c_int, _P]
lib.negf_rgf_lesser_greater.argtypes = [_P, C.POINTER(Problem), C.POINTER(Sigma), C.POINTER(Sigma),
                                        C.POINTER(Sigma), _P, _P, _P, _P, _P, _P]
lib.negf_observables.argtypes = [_P, C.POINTER(Problem)] + [_P] * 19
lib.negf_energy_convolve.argtypes = [_P, C.c_int, C.c_longlong, C.c_int, _P, _P, C.c_int, C.c_int, c128, _P]
lib.negf_pipeline_host_bytes.argtypes = [C.POINTER(Problem), C.c_int, C.c_int, C.POINTER(C.c_size_t)]
lib.negf_pipeline_device.argtypes = [_P, C.POINTER(Problem), C.POINTER(Sigma), C.POINTER(Sigma), C.POINTER(Sigma), _P,
                                     C.c_double, C.c_double, C.c_double, C.c_double, C.c_int, C.POINTER(DeviceOutputs)]
lib.negf_pipeline_host.argtypes = [_P, C.POINTER(Problem), C.POINTER(Sigma), C.POINTER(Sigma), C.POINTER(Sigma),
                                   _P, C.c_double, C.c_double, C.c_double, C.c_double, C.c_int, _P, C.c_size_t,
                                   C.POINTER(HostOutputs), C.POINTER(C.c_size_t), C.POINTER(C.c_size_t)]
lib.negf_zgemm_batched.argtypes = [_P, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, c128, _P, C.c_int,
                                   C.c_longlong, _P, C.c_int, C.c_longlong, c128, _P, _P, C.c_int,
                                   C.c_longlong, C.c_int]
lib.negf_zinverse_batched.argtypes = [_P, C.c_int, _P, C.c_longlong, C.c_int, _P]
lib.negf_zinverse_batched_static.argtypes = [_P, C.c_int, _P, C.c_longlong, C.c_int, _P]
lib.negf_fp64_peak.argtypes = [_P, C.c_double, C.POINTER(C.c_double)]


class NegfError(RuntimeError):
    pass


def strerror(code: int) -> str:
    return lib.negf_strerror(code).decode()


def _ptr(t) -> Optional[int]:
    """Device (or host) address of a tensor / numpy array / None."""
    if t is None:
        return None
    if hasattr(t, "data_ptr"):
        if not t.is_contiguous():
            raise ValueError("tensor must be contiguous")
        return t.data_ptr()
    if hasattr(t, "ctypes"):
        if not t.flags["C_CONTIGUOUS"]:
            raise ValueError("array must be C-contiguous")
        return t.ctypes.data
    return int(t)


def make_problem(n_blocks, block_size, n_energy, H_diag, H_upper, S_diag, S_upper, energy, eta,
                 n_k: int = 1, k_index=None) -> Problem:
    """n_k > 1: H / S arrays are [n_k][...] and k_index [n_energy] (int32) names the device of every batch entry."""
    return Problem(n_blocks, block_size, n_energy, _ptr(H_diag), _ptr(H_upper), _ptr(S_diag), _ptr(S_upper),
                   _ptr(energy), float(eta), int(n_k), _ptr(k_index))


def make_sigma(kind=SIGMA_NONE, scalar=None, diag=None, upper=None, lower=None, left=None, right=None) -> Sigma:
    return Sigma(kind, _ptr(scalar), _ptr(diag), _ptr(upper), _ptr(lower), _ptr(left), _ptr(right))


class Context:
    """negf_ctx*.  Methods carry the C names without the negf_ prefix."""

    def __init__(self, device: int = 0):
        h = _P()
        rc = lib.negf_create(C.byref(h), device)
        if rc != OK:
            raise NegfError(f"negf_create: {strerror(rc)} (no CPU fallback exists)")
        self._h = h
        self._ws = None

    def _check(self, rc, what):
        if rc != OK:
            extra = f" [cudaError {lib.negf_last_cuda_error(self._h)}]" if rc == ECUDA else ""
            raise NegfError(f"{what}: {strerror(rc)}{extra}")

    def close(self):
        if self._h:
            lib.negf_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_stream(self, cuda_stream: int):
        self._check(lib.negf_set_stream(self._h, cuda_stream), "negf_set_stream")

    @staticmethod
    def workspace_bytes(p: Problem, kind_max: int = SIGMA_BT, flags: int = KEEP_SWEEP) -> int:
        out = C.c_size_t()
        rc = lib.negf_workspace_bytes(C.byref(p), kind_max, flags, C.byref(out))
        if rc != OK:
            raise NegfError(f"negf_workspace_bytes: {strerror(rc)}")
        return out.value

    def set_workspace(self, tensor):
        """tensor: a torch uint8 CUDA tensor owned by the caller (kept alive here)."""
        self._ws = tensor
        self._check(lib.negf_set_workspace(self._h, _ptr(tensor), 0 if tensor is None else tensor.numel()),
                    "negf_set_workspace")

    def set_option(self, option: int, value: int):
        self._check(lib.negf_set_option(self._h, option, value), "negf_set_option")

    def launch_count(self) -> int:
        return int(lib.negf_launch_count(self._h))

    def obc_graph_kernels(self) -> int:
        return int(lib.negf_obc_graph_kernels(self._h))

    def profile_enable(self, on: bool):
        self._check(lib.negf_profile_enable(self._h, int(on)), "negf_profile_enable")

    def profile_read(self, kclass: int, reset: bool = True):
        """(milliseconds, launch sites) of one kernel class since the last reset; synchronises."""
        ms, n = C.c_double(), C.c_longlong()
        self._check(lib.negf_profile_read(self._h, kclass, C.byref(ms), C.byref(n), int(reset)), "negf_profile_read")
        return ms.value, n.value

    def obc_decimate(self, p: Problem, side, mu, kT, tol, max_iter, sigma_r, gamma=None, sigma_lesser=None,
                     sigma_greater=None, g_surface=None, fermi=None, iters=None, status=None, lead: Lead = None):
        self._check(lib.negf_obc_decimate(self._h, C.byref(p), C.byref(lead) if lead is not None else None,
                                          side, mu, kT, tol, max_iter, _ptr(sigma_r), _ptr(gamma),
                                          _ptr(sigma_lesser), _ptr(sigma_greater), _ptr(g_surface), _ptr(fermi),
                                          _ptr(iters), _ptr(status)), "negf_obc_decimate")

    def obc_decimate_pair(self, p: Problem, mu_L, mu_R, kT, tol, max_iter, left: dict, right: dict,
                          lead_L: Lead = None, lead_R: Lead = None):
        """left / right: dicts with the keys of negf_obc_out (tensors or None)."""
        keys = ("sigma_r", "gamma", "sigma_lesser", "sigma_greater", "g_surface", "fermi", "iters", "status")
        oL = ObcOut(*[_ptr(left.get(k)) for k in keys])
        oR = ObcOut(*[_ptr(right.get(k)) for k in keys])
        ref = lambda s: C.byref(s) if s is not None else None
        self._check(lib.negf_obc_decimate_pair(self._h, C.byref(p), ref(lead_L), ref(lead_R), mu_L, mu_R, kT, tol,
                                               max_iter, C.byref(oL), C.byref(oR)), "negf_obc_decimate_pair")

    def rgf_retarded(self, p: Problem, sigma_r: Optional[Sigma], GR_diag, GR_upper=None, GR_lower=None,
                     GR_corner=None, flags=0, info=None):
        self._check(lib.negf_rgf_retarded(self._h, C.byref(p), C.byref(sigma_r) if sigma_r is not None else None,
                                          _ptr(GR_diag), _ptr(GR_upper), _ptr(GR_lower), _ptr(GR_corner), flags,
                                          _ptr(info)), "negf_rgf_retarded")

    def rgf_lesser_greater(self, p: Problem, sigma_r, sigma_lesser, sigma_greater, GR_diag, GL_diag=None,
                           GL_upper=None, GG_diag=None, GG_upper=None, info=None):
        ref = lambda s: C.byref(s) if s is not None else None
        self._check(lib.negf_rgf_lesser_greater(self._h, C.byref(p), ref(sigma_r), ref(sigma_lesser),
                                                ref(sigma_greater), _ptr(GR_diag), _ptr(GL_diag), _ptr(GL_upper),
                                                _ptr(GG_diag), _ptr(GG_upper), _ptr(info)),
                    "negf_rgf_lesser_greater")

    def observables(self, p: Problem, GR_diag=None, GR_upper=None, GR_lower=None, GR_corner=None, GL_diag=None,
                    GL_upper=None, GG_diag=None, gamma_L=None, gamma_R=None, sigma_lesser_L=None,
                    sigma_greater_L=None, sigma_lesser_R=None, sigma_greater_R=None, weights=None, density=None,
                    ldos=None, transmission=None, bond_current=None, contact_current=None):
        args = [GR_diag, GR_upper, GR_lower, GR_corner, GL_diag, GL_upper, GG_diag, gamma_L, gamma_R,
                sigma_lesser_L, sigma_greater_L, sigma_lesser_R, sigma_greater_R, weights, density, ldos,
                transmission, bond_current, contact_current]
        self._check(lib.negf_observables(self._h, C.byref(p), *[_ptr(a) for a in args]), "negf_observables")

    def energy_convolve(self, n_energy, elems_per_energy, X1, X2, Y, mode=0, conj2=False, scale=1.0, transpose_block=0):
        sc = complex(scale)
        self._check(lib.negf_energy_convolve(self._h, n_energy, elems_per_energy, transpose_block, _ptr(X1), _ptr(X2),
                                             mode, int(conj2), c128(sc.real, sc.imag), _ptr(Y)), "negf_energy_convolve")

    def pipeline_device(self, p: Problem, sigma_r, sigma_lesser, sigma_greater, weights, mu_L, mu_R, kT, tol, max_iter,
                        outputs: DeviceOutputs):
        ref = lambda s: C.byref(s) if s is not None else None
        self._check(lib.negf_pipeline_device(self._h, C.byref(p), ref(sigma_r), ref(sigma_lesser), ref(sigma_greater),
                                             _ptr(weights), mu_L, mu_R, kT, tol, max_iter, C.byref(outputs)),
                    "negf_pipeline_device")

    @staticmethod
    def pipeline_host_bytes(p: Problem, kind_max: int, want_greater: bool) -> int:
        out = C.c_size_t()
        rc = lib.negf_pipeline_host_bytes(C.byref(p), kind_max, int(want_greater), C.byref(out))
        if rc != OK:
            raise NegfError(f"negf_pipeline_host_bytes: {strerror(rc)}")
        return out.value

    def pipeline_host(self, host_problem: Problem, sigma_r, sigma_lesser, sigma_greater, weights, mu_L, mu_R, kT,
                      tol, max_iter, dev_scratch, outputs: HostOutputs):
        ref = lambda s: C.byref(s) if s is not None else None
        up, down = C.c_size_t(), C.c_size_t()
        self._check(lib.negf_pipeline_host(self._h, C.byref(host_problem), ref(sigma_r), ref(sigma_lesser),
                                           ref(sigma_greater), _ptr(weights), mu_L, mu_R, kT, tol, max_iter,
                                           _ptr(dev_scratch), dev_scratch.numel(), C.byref(outputs),
                                           C.byref(up), C.byref(down)), "negf_pipeline_host")
        return up.value, down.value

    def zgemm_batched(self, opA, opB, m, n, k, alpha, A, lda, strideA, B, ldb, strideB, beta, D, Cout, ldc,
                      strideC, batch):
        al, be = complex(alpha), complex(beta)
        self._check(lib.negf_zgemm_batched(self._h, opA, opB, m, n, k, c128(al.real, al.imag), _ptr(A), lda,
                                           strideA, _ptr(B), ldb, strideB, c128(be.real, be.imag), _ptr(D),
                                           _ptr(Cout), ldc, strideC, batch), "negf_zgemm_batched")

    def zinverse_batched(self, b, A, stride, batch, info=None):
        self._check(lib.negf_zinverse_batched(self._h, b, _ptr(A), stride, batch, _ptr(info)),
                    "negf_zinverse_batched")

    def zinverse_batched_static(self, b, A, stride, batch, info=None):
        """No-allocation variant: scratch in the library's static device array (include/negf.h)."""
        self._check(lib.negf_zinverse_batched_static(self._h, b, _ptr(A), stride, batch, _ptr(info)),
                    "negf_zinverse_batched_static")

    def fp64_peak(self, ms: float = 200.0) -> float:
        out = C.c_double()
        self._check(lib.negf_fp64_peak(self._h, ms, C.byref(out)), "negf_fp64_peak")
        return out.value
