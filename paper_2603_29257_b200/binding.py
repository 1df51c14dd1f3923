"""ctypes binding of include/risp.h -- argument marshalling only."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None

EXPORTED_SYMBOLS = ["risp_setup", "risp_matvec", "risp_matvec_host", "risp_tda_solve", "risp_destroy", "risp_last_error",
                    "risp_get_dims", "risp_get_timings", "risp_eri3c_shell", "risp_get_stage", "risp_transition_properties", "risp_matvec_tddft", "risp_tddft_solve", "risp_matvec_shard_begin", "risp_matvec_shard_end"]

RISP_MAX_ROOTS = 64
FLAG_KEEP_STAGES, FLAG_SPILL_HALF, FLAG_SMALL_KBUILD, FLAG_TDDFT = 1, 2, 4, 8
SOLVE_NO_CACHE, SOLVE_TINY_CACHE, SOLVE_PERTURBED_GUESS, SOLVE_HOST_FP32 = 1, 2, 4, 8
STAGE = dict(R=1, RTILDE=2, J=3, K=4, TIJ=5, TAB=6, PAIRS=7, METRIC_J=8, METRIC_K=9, U=10)
_ERR = {-1: "RISP_EINVAL", -2: "RISP_ENOMEM", -3: "RISP_ECUDA", -4: "RISP_ENOTPD", -5: "RISP_ENOTCONV"}


class RispError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{_ERR.get(code, code)}: {msg}")
        self.code = code


class _System(C.Structure):
    _fields_ = [("natm", C.c_int32), ("xyz_bohr", C.POINTER(C.c_double)), ("Z", C.POINTER(C.c_int32)),
                ("nshl", C.c_int32), ("shl_atom", C.POINTER(C.c_int32)), ("shl_l", C.POINTER(C.c_int32)),
                ("shl_nprim", C.POINTER(C.c_int32)), ("shl_poff", C.POINTER(C.c_int32)),
                ("prim_exp", C.POINTER(C.c_double)), ("prim_coef", C.POINTER(C.c_double)),
                ("naux", C.c_int32), ("aux_atom", C.POINTER(C.c_int32)), ("aux_l", C.POINTER(C.c_int32)),
                ("aux_exp", C.POINTER(C.c_double)), ("aux_in_K", C.POINTER(C.c_uint8)),
                ("nao", C.c_int32), ("nocc", C.c_int32), ("nvir", C.c_int32),
                ("C", C.POINTER(C.c_double)), ("eps", C.POINTER(C.c_double)),
                ("alpha", C.c_double), ("beta", C.c_double), ("omega", C.c_double), ("cutoff_ev", C.c_double)]


class _Options(C.Structure):
    _fields_ = [("screen_tol", C.c_double), ("hbm_budget_bytes", C.c_size_t), ("host_budget_bytes", C.c_size_t),
                ("device", C.c_int32), ("flags", C.c_int32), ("max_batch", C.c_int32), ("reserved", C.c_int32),
                ("shard_rank", C.c_int32), ("shard_count", C.c_int32)]


class _SolveOptions(C.Structure):
    _fields_ = [("tol", C.c_double), ("max_iter", C.c_int32), ("n_guess", C.c_int32), ("max_sub", C.c_int32), ("flags", C.c_int32),
                ("max_block", C.c_int32), ("max_seconds", C.c_int32), ("device_budget_bytes", C.c_size_t)]


class _SolveInfo(C.Structure):
    _fields_ = [("iterations", C.c_int32), ("restarts", C.c_int32), ("n_sigma", C.c_int32), ("converged", C.c_int32),
                ("resid", C.c_double * RISP_MAX_ROOTS), ("sec_total", C.c_double), ("sec_matvec", C.c_double),
                ("sec_subspace", C.c_double), ("bytes_h2d", C.c_double), ("bytes_d2h", C.c_double), ("subspace_max", C.c_int32), ("cached_vectors", C.c_int32), ("sec_alloc", C.c_double),
                ("block", C.c_int32), ("capacity", C.c_int32), ("bytes_host_subspace", C.c_double)]


class _Dims(C.Structure):
    _fields_ = [("nao", C.c_int32), ("nocc", C.c_int32), ("nvir", C.c_int32), ("nauxJ", C.c_int32), ("nauxK", C.c_int32),
                ("noccK", C.c_int32), ("nvirK", C.c_int32), ("occK_first", C.c_int32), ("virK_first", C.c_int32),
                ("n_shell_pairs", C.c_int64), ("n_shell_pairs_kept", C.c_int64), ("n_ao_pairs_kept", C.c_int64),
                ("bytes_Tij", C.c_int64), ("bytes_Tab", C.c_int64), ("bytes_device_total", C.c_int64), ("aux_chunk", C.c_int32),
                ("nauxK_device", C.c_int32), ("bytes_T_host", C.c_int64), ("j_sub_batch", C.c_int32), ("j_panels", C.c_int32),
                ("pairs_per_class", C.c_int64 * 6), ("n_aux_centres", C.c_int64)]


class _Timings(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("total", "j_transform_in", "j_pass1", "j_solve", "j_pass2", "j_transform_out",
                                          "k_gather", "k_gemm1", "k_gemm2", "k_total", "assemble")] + \
               [("kernel_launches", C.c_int32), ("first_chunk_naux", C.c_int32)]


def library_path() -> str:
    return os.path.join(_HERE, "librisp.so")


def load_library():
    """dlopen librisp.so (built in-tree by paper_2603_29257_b200.build).  Fails loudly if it is missing."""
    global _LIB
    if _LIB is not None:
        return _LIB
    path = library_path()
    if not os.path.exists(path):
        raise RispError(-3, f"{path} not found: run `python -m paper_2603_29257_b200.build` (no CPU fallback exists)")
    lib = C.CDLL(path)
    vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
    lib.risp_setup.argtypes = [C.POINTER(_System), C.POINTER(_Options), C.POINTER(vp)]
    lib.risp_matvec.argtypes = [vp, i32, vp, vp, vp]
    lib.risp_matvec_host.argtypes = [vp, i32, vp, vp]
    lib.risp_tda_solve.argtypes = [vp, i32, C.POINTER(_SolveOptions), C.POINTER(dbl), vp, C.POINTER(_SolveInfo)]
    lib.risp_destroy.argtypes = [vp]; lib.risp_destroy.restype = None
    lib.risp_last_error.argtypes = [vp]; lib.risp_last_error.restype = C.c_char_p
    lib.risp_get_dims.argtypes = [vp, C.POINTER(_Dims)]
    lib.risp_get_timings.argtypes = [vp, C.POINTER(_Timings)]
    lib.risp_eri3c_shell.argtypes = [vp, i32, i32, i32, i32, vp]
    lib.risp_get_stage.argtypes = [vp, i32, vp, i64, vp]
    lib.risp_set_precision.argtypes = [vp, i32]
    lib.risp_matvec_shard_begin.argtypes = [vp, i32, vp, vp, vp]
    lib.risp_matvec_shard_end.argtypes = [vp, i32, vp, vp, vp, vp]
    lib.risp_matvec_tddft.argtypes = [vp, i32, vp, vp, vp, vp]
    lib.risp_tddft_solve.argtypes = [vp, i32, C.POINTER(_SolveOptions), C.POINTER(dbl), vp, vp, C.POINTER(_SolveInfo)]
    lib.risp_transition_properties.argtypes = [vp, i32, vp, vp, vp, dbl, vp, vp, vp, vp]
    # include/risp_debug.h
    lib.risp_debug_oneel_ao.argtypes = [vp, vp, vp]
    lib.risp_debug_dgemm.argtypes = [C.c_int, C.c_int, C.c_int, vp, C.c_longlong, C.c_int, vp, C.c_longlong, C.c_int, vp, C.c_longlong,
                                     dbl, dbl, C.c_int, C.c_longlong, C.c_longlong, C.c_longlong, C.c_int, C.c_int, C.c_longlong, vp]
    lib.risp_debug_tcgemm.argtypes = [C.c_int32, C.c_int32, C.c_int32, C.c_int32, vp, vp, vp, C.c_int32, C.c_int32, C.c_int32, C.c_int32, vp]
    lib.risp_debug_set_tc_plan.argtypes = [vp, C.c_int32, C.c_int32, C.c_int32, C.c_int32]
    lib.risp_tcgemm_static.argtypes = [C.c_int32, C.c_int32, C.c_int32, vp, vp, vp, C.c_int32, vp]
    lib.risp_static_last_error.restype = C.c_char_p
    lib.risp_debug_sym_eig_lowest.argtypes = [C.c_int, C.c_int, vp, vp, vp]
    lib.risp_debug_force_plan.argtypes = [vp, C.c_int, C.c_int, C.c_int]
    lib.risp_debug_yardstick.argtypes = [vp, C.c_int, C.c_size_t, C.c_int, C.POINTER(dbl)]
    _LIB = lib
    return lib


def _struct_dict(s):
    out = {}
    for name, _ in s._fields_:
        v = getattr(s, name)
        out[name] = list(v) if hasattr(v, "__len__") else v
    return out


class RispContext:
    """Owns one `risp_ctx`.  X / sigma are torch CUDA tensors (device pointers go straight through the ABI)."""

    def __init__(self, sys: dict, screen_tol: float = 0.0, hbm_budget_bytes: int = 0, host_budget_bytes: int = 0, device: int = 0,
                 flags: int = 0, max_batch: int = 0, shard_rank: int = 0, shard_count: int = 0):
        self.lib = load_library()
        keep = {}

        def arr(key, dt):
            a = np.ascontiguousarray(sys[key], dtype=dt)
            keep[key] = a
            return a.ctypes.data_as(C.POINTER({np.float64: C.c_double, np.int32: C.c_int32, np.uint8: C.c_uint8}[dt]))

        s = _System()
        s.natm = int(sys["natm"]); s.xyz_bohr = arr("xyz_bohr", np.float64); s.Z = arr("Z", np.int32)
        s.nshl = int(sys["nshl"])
        for k in ("shl_atom", "shl_l", "shl_nprim", "shl_poff"):
            setattr(s, k, arr(k, np.int32))
        s.prim_exp = arr("prim_exp", np.float64); s.prim_coef = arr("prim_coef", np.float64)
        s.naux = int(sys["naux"]); s.aux_atom = arr("aux_atom", np.int32); s.aux_l = arr("aux_l", np.int32)
        s.aux_exp = arr("aux_exp", np.float64); s.aux_in_K = arr("aux_in_K", np.uint8)
        s.nao, s.nocc, s.nvir = int(sys["nao"]), int(sys["nocc"]), int(sys["nvir"])
        s.C = arr("C", np.float64); s.eps = arr("eps", np.float64)
        s.alpha, s.beta, s.omega, s.cutoff_ev = float(sys["alpha"]), float(sys["beta"]), float(sys["omega"]), float(sys["cutoff_ev"])
        o = _Options(float(screen_tol), int(hbm_budget_bytes), int(host_budget_bytes), int(device), int(flags), int(max_batch), 0, int(shard_rank), int(shard_count))
        self.handle = C.c_void_p()
        self.nocc, self.nvir, self.nao = s.nocc, s.nvir, s.nao
        self.device = device
        rc = self.lib.risp_setup(C.byref(s), C.byref(o), C.byref(self.handle))
        if rc != 0:
            msg = self.lib.risp_last_error(self.handle).decode()
            self.close()
            raise RispError(rc, msg)
        self.aux_l = np.asarray(sys["aux_l"]); self.shl_l = np.asarray(sys["shl_l"])

    def _check(self, rc):
        if rc != 0:
            raise RispError(rc, self.lib.risp_last_error(self.handle).decode())

    def close(self):
        if getattr(self, "handle", None) is not None and self.handle:
            self.lib.risp_destroy(self.handle)
        self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- hot path
    def matvec(self, X, sigma=None, stream=None):
        import torch
        assert X.is_cuda and X.dtype == torch.float64 and X.is_contiguous()
        m = X.shape[0]
        if sigma is None:
            sigma = torch.empty_like(X)
        st = torch.cuda.current_stream(X.device).cuda_stream if stream is None else stream
        self._check(self.lib.risp_matvec(self.handle, m, X.data_ptr(), sigma.data_ptr(), st))
        return sigma

    def matvec_host(self, X: np.ndarray, sigma: np.ndarray | None = None) -> np.ndarray:
        X = np.ascontiguousarray(X, dtype=np.float64)
        if sigma is None:
            sigma = np.empty_like(X)
        self._check(self.lib.risp_matvec_host(self.handle, X.shape[0], X.ctypes.data, sigma.ctypes.data))
        return sigma

    def matvec_host_ptr(self, m: int, x_ptr: int, s_ptr: int):
        """Host buffers given as raw addresses (e.g. pinned torch tensors)."""
        self._check(self.lib.risp_matvec_host(self.handle, m, x_ptr, s_ptr))

    def tda_solve(self, nroots, tol=1e-5, max_iter=100, n_guess=0, max_sub=0, want_vectors=False, allow_unconverged=False, flags=0,
                  max_block=0, device_budget_bytes=0, max_seconds=0):
        import torch
        omega = np.zeros(nroots)
        info = _SolveInfo()
        opt = _SolveOptions(float(tol), int(max_iter), int(n_guess), int(max_sub), int(flags), int(max_block), int(max_seconds), int(device_budget_bytes))
        if want_vectors and (flags & 16):      # RISP_SOLVE_X_OUT_HOST: a host array takes the vectors
            X = np.empty((nroots, self.nocc, self.nvir))
            xptr = X.ctypes.data
        else:
            X = torch.empty((nroots, self.nocc, self.nvir), dtype=torch.float64, device=f"cuda:{self.device}") if want_vectors else None
            xptr = X.data_ptr() if X is not None else None
        rc = self.lib.risp_tda_solve(self.handle, nroots, C.byref(opt), omega.ctypes.data_as(C.POINTER(C.c_double)), xptr, C.byref(info))
        if rc != 0 and not (rc == -5 and allow_unconverged):
            self._check(rc)
        d = _struct_dict(info)
        d["resid"] = d["resid"][:nroots]
        return omega, X, d

    def matvec_shard_begin(self, X, R=None, stream=None):
        """first half of a P-sharded sigma-build: this rank's partial R_mQ as a [nauxJ][32] device tensor"""
        import torch
        if R is None:
            R = torch.empty((self.dims()["nauxJ"], 32), dtype=torch.float64, device=X.device)
        st = torch.cuda.current_stream(X.device).cuda_stream if stream is None else stream
        self._check(self.lib.risp_matvec_shard_begin(self.handle, X.shape[0], X.data_ptr(), R.data_ptr(), st))
        return R

    def matvec_shard_end(self, X, R, sigma=None, stream=None):
        import torch
        if sigma is None:
            sigma = torch.empty_like(X)
        st = torch.cuda.current_stream(X.device).cuda_stream if stream is None else stream
        self._check(self.lib.risp_matvec_shard_end(self.handle, X.shape[0], X.data_ptr(), R.data_ptr(), sigma.data_ptr(), st))
        return sigma

    def matvec_tddft(self, X, stream=None):
        """risp_matvec_tddft: ((A+B) X, (A-B) X) for the device vectors X[m][nocc][nvir]."""
        import torch
        assert X.is_cuda and X.dtype == torch.float64 and X.is_contiguous()
        sp, sm = torch.empty_like(X), torch.empty_like(X)
        st = torch.cuda.current_stream(X.device).cuda_stream if stream is None else stream
        self._check(self.lib.risp_matvec_tddft(self.handle, X.shape[0], X.data_ptr(), sp.data_ptr(), sm.data_ptr(), st))
        return sp, sm

    def tddft_solve(self, nroots, tol=1e-5, max_iter=100, n_guess=0, max_sub=0, want_vectors=False, allow_unconverged=False, device_budget_bytes=0):
        import torch
        omega = np.zeros(nroots)
        info = _SolveInfo()
        opt = _SolveOptions(float(tol), int(max_iter), int(n_guess), int(max_sub), 0, 0, 0, int(device_budget_bytes))
        X = Y = None
        if want_vectors:
            X = torch.empty((nroots, self.nocc, self.nvir), dtype=torch.float64, device=f"cuda:{self.device}")
            Y = torch.empty_like(X)
        rc = self.lib.risp_tddft_solve(self.handle, nroots, C.byref(opt), omega.ctypes.data_as(C.POINTER(C.c_double)),
                                       X.data_ptr() if X is not None else None, Y.data_ptr() if Y is not None else None, C.byref(info))
        if rc != 0 and not (rc == -5 and allow_unconverged):
            self._check(rc)
        d = _struct_dict(info)
        d["resid"] = d["resid"][:nroots]
        return omega, X, Y, d

    def transition_properties(self, X, omega, origin=None, scale=0.0):
        """risp_transition_properties: (mu[n][3], m[n][3], f[n], R[n]) for the device vectors X[n][nocc][nvir]."""
        n = X.shape[0]
        om = np.ascontiguousarray(omega, dtype=np.float64)
        org = None if origin is None else np.ascontiguousarray(origin, dtype=np.float64)
        mu, m, f, R = np.zeros((n, 3)), np.zeros((n, 3)), np.zeros(n), np.zeros(n)
        self._check(self.lib.risp_transition_properties(self.handle, n, X.data_ptr(), om.ctypes.data, org.ctypes.data if org is not None else None,
                                                        float(scale), mu.ctypes.data, m.ctypes.data, f.ctypes.data, R.ctypes.data))
        return mu, m, f, R

    def oneel_ao(self, origin=None) -> np.ndarray:
        org = None if origin is None else np.ascontiguousarray(origin, dtype=np.float64)
        out = np.zeros((6, self.nao, self.nao))
        self._check(self.lib.risp_debug_oneel_ao(self.handle, org.ctypes.data if org is not None else None, out.ctypes.data))
        return out

    def set_precision(self, mode: int):
        """0: FP64 (default); 1: the K contractions in the paper's single precision on the tcgen05 tensor cores; 2: as 1, and the
        AO<->MO transforms of the J term as well (RISP_PRECISION_FP32_JK)."""
        self._check(self.lib.risp_set_precision(self.handle, int(mode)))

    def force_plan(self, mj: int = 0, prow: int = 0, pc: int = 0):
        """Testing: override the work-space plan (J sub-batch, AO rows per panel, K aux chunk); 0 keeps the automatic choice."""
        self._check(self.lib.risp_debug_force_plan(self.handle, mj, prow, pc))

    def yardstick(self, which: int, nbytes: int = 0, reps: int = 5) -> float:
        """risp_debug_yardstick: 0 DFMA flop/s, 1 DMMA flop/s, 2 device copy bytes/s (read + write)."""
        out = C.c_double(0.0)
        self._check(self.lib.risp_debug_yardstick(self.handle, which, nbytes, reps, C.byref(out)))
        return out.value

    # ---- getters
    def dims(self) -> dict:
        d = _Dims()
        self._check(self.lib.risp_get_dims(self.handle, C.byref(d)))
        return _struct_dict(d)

    def timings(self) -> dict:
        t = _Timings()
        self._check(self.lib.risp_get_timings(self.handle, C.byref(t)))
        return _struct_dict(t)

    def eri3c_shell(self, si, sj, ak, op=0) -> np.ndarray:
        out = np.zeros((2 * int(self.shl_l[si]) + 1, 2 * int(self.shl_l[sj]) + 1, 2 * int(self.aux_l[ak]) + 1))
        self._check(self.lib.risp_eri3c_shell(self.handle, si, sj, ak, op, out.ctypes.data))
        return out

    def stage(self, which: str, m: int = 0, sel=None) -> np.ndarray:
        d = self.dims()
        shape = {"R": (d["nauxJ"], m), "RTILDE": (d["nauxJ"], m), "J": (m, d["nocc"], d["nvir"]), "K": (m, d["nocc"], d["nvir"]),
                 "TIJ": (len(sel) if sel is not None else 0, d["noccK"], d["noccK"]),
                 "TAB": (len(sel) if sel is not None else 0, d["nvirK"], d["nvirK"]),
                 "PAIRS": (d["n_shell_pairs_kept"], 2), "METRIC_J": (d["nauxJ"], d["nauxJ"]), "METRIC_K": (d["nauxK"], d["nauxK"]),
                 "U": (d["nao"], d["nao"])}[which]
        out = np.zeros(shape, dtype=np.int64 if which == "PAIRS" else np.float64)
        selarr = np.ascontiguousarray(sel, dtype=np.int64) if sel is not None else None
        self._check(self.lib.risp_get_stage(self.handle, STAGE[which], selarr.ctypes.data if selarr is not None else None,
                                            len(selarr) if selarr is not None else 0, out.ctypes.data))
        return out


def setup(sys: dict, **kw) -> RispContext:
    """risp_setup: build pair list, metrics, window and K tensors for `sys` (fields of `risp_system`)."""
    return RispContext(sys, **kw)


STATIC_SCRATCH_BYTES = 16 << 20


def tcgemm_static(A, B, C_out=None, accumulate=False, stream=None):
    """`risp_tcgemm_static`: C[c][r] (+)= sum_k A[r][k] B[c][k] in the single-precision mode, allocating nothing inside the library
    (A [M][K], B [N][K], C [N][M]: contiguous FP64 torch CUDA tensors; C_out is created here, by torch, when not given)."""
    import torch
    lib = load_library()
    M, K = A.shape
    N = B.shape[0]
    if C_out is None:
        C_out = torch.empty((N, M), dtype=torch.float64, device=A.device)
    st = C.c_void_p(stream.cuda_stream) if stream is not None else C.c_void_p(torch.cuda.current_stream(A.device).cuda_stream)
    rc = lib.risp_tcgemm_static(M, N, K, A.data_ptr(), B.data_ptr(), C_out.data_ptr(), 1 if accumulate else 0, st)
    if rc != 0:
        raise RispError(rc, lib.risp_static_last_error().decode())
    return C_out
