"""Thin ctypes binding of the C ABI in ``include/gmmnlse.h`` (same names, argument marshalling only).

Every step of the path runs in the CUDA kernels behind ``libgmmnlse.so``; there is no CPU or
PyTorch fallback: if the library is missing this module raises.  torch is used for device memory
and streams only (tensors are passed as ``data_ptr()``).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

OK, WARN_NOCONV, EINVAL, ENOMEM, ECUDA, EUNSUPPORTED = 0, 1, -1, -2, -3, -4


KINDS = ("fft_to_time", "pair_conv", "contract", "mode_reduce", "fft_to_freq", "scan", "advance", "misc")


class GmmnlseError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"gmmnlse status {status}: {msg}")
        self.status = status


class Options(C.Structure):
    _fields_ = [("precision", C.c_int), ("shock", C.c_int), ("tol", C.c_double), ("max_iter", C.c_int),
                ("fixed_iter", C.c_int), ("contraction", C.c_int), ("raman", C.c_int), ("graph", C.c_int),
                ("stop_rule", C.c_int), ("async_call", C.c_int)]


_LIB = None
_DP = C.POINTER(C.c_double)
_LLP = C.POINTER(C.c_longlong)

# name -> (restype, argtypes): every symbol include/gmmnlse.h declares
SIGNATURES = {
    "gmmnlse_plan_create": (C.c_int, [C.POINTER(C.c_void_p), C.c_int, C.c_int, C.c_int, C.c_double, C.c_double,
                                      _DP, C.c_int, _DP, C.c_double, _DP, C.c_double, C.c_double,
                                      C.POINTER(Options)]),
    "gmmnlse_plan_create_general": (C.c_int, [C.POINTER(C.c_void_p), C.c_int, C.c_int, C.c_int, C.c_double,
                                              C.c_double, _DP, C.c_int, _DP, _DP, C.c_int, C.c_double, _DP,
                                              C.c_double, C.c_double, C.POINTER(Options)]),
    "gmmnlse_propagate": (C.c_int, [C.c_void_p, C.c_void_p, C.c_double, C.c_void_p, C.c_void_p]),
    "gmmnlse_propagate_host": (C.c_int, [C.c_void_p, C.c_void_p, C.c_double, C.c_void_p]),
    "gmmnlse_propagate_rk4ip": (C.c_int, [C.c_void_p, C.c_void_p, C.c_double, C.c_void_p, C.c_void_p]),
    "gmmnlse_nonlinear_op": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "gmmnlse_shard_begin": (C.c_int, [C.c_void_p, C.c_void_p]),
    "gmmnlse_shard_iterate": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p]),
    "gmmnlse_shard_update": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_int, C.c_int,
                                       _DP]),
    "gmmnlse_shard_advance": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p, C.c_int]),
    "gmmnlse_shard_end": (C.c_int, [C.c_void_p, C.c_void_p]),
    "gmmnlse_set_gain": (C.c_int, [C.c_void_p, _DP]),
    "gmmnlse_set_coupling": (C.c_int, [C.c_void_p, _DP]),
    "gmmnlse_set_coupling_profile": (C.c_int, [C.c_void_p, _DP, C.c_int]),
    "gmmnlse_set_gain_saturation": (C.c_int, [C.c_void_p, C.c_double]),
    "gmmnlse_set_stream": (C.c_int, [C.c_void_p, C.c_void_p]),
    "gmmnlse_get_stats": (C.c_int, [C.c_void_p, _LLP, _LLP, _DP, _LLP]),
    "gmmnlse_launch_count": (C.c_longlong, [C.c_void_p]),
    "gmmnlse_profile_enable": (C.c_int, [C.c_void_p, C.c_int]),
    "gmmnlse_profile_get": (C.c_int, [C.c_void_p, C.c_int, _DP, _LLP]),
    "gmmnlse_debug_get_planes": (C.c_int, [C.c_void_p, C.c_void_p]),
    "gmmnlse_debug_fft": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int]),
    "gmmnlse_debug_pairs": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]),
    "gmmnlse_debug_contract": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]),
    "gmmnlse_contraction_kind": (C.c_int, [C.c_void_p]),
    "gmmnlse_raman_kind": (C.c_int, [C.c_void_p]),
    "gmmnlse_lowrank_rank": (C.c_int, [C.c_void_p]),
    "gmmnlse_sparse_info": (C.c_int, [C.c_void_p, C.POINTER(C.c_int), _DP]),
    "gmmnlse_loop_kind": (C.c_int, [C.c_void_p]),
    "gmmnlse_debug_set_tc_chunk": (C.c_int, [C.c_void_p, C.c_int]),
    "gmmnlse_overlap_tensor": (C.c_int, [C.c_int, C.c_longlong, _DP, C.c_double, _DP]),
    "gmmnlse_overlap_tensor_noalloc": (C.c_int, [C.c_int, C.c_longlong, C.c_void_p, C.c_double, C.c_void_p, C.c_void_p]),
    "gmmnlse_overlap_tensor_noalloc_limits": (C.c_int, [C.POINTER(C.c_int), _LLP, _LLP]),
    "gmmnlse_plan_destroy": (None, [C.c_void_p]),
    "gmmnlse_status_string": (C.c_char_p, [C.c_int]),
    "gmmnlse_last_cuda_error": (C.c_char_p, []),
    "gmmnlse_abi_version": (C.c_int, []),
}


def load_library(path: str | None = None):
    """dlopen ``libgmmnlse.so`` (built in-tree by ``build.build()``); raises if it is absent."""
    global _LIB
    if _LIB is not None and path is None:
        return _LIB
    path = path or _build.LIB_PATH
    if not os.path.exists(path):
        raise GmmnlseError(ECUDA, f"{path} not built: run `python -m paper_1708_05324_b200.build` "
                                  "(no CPU fallback exists)")
    lib = C.CDLL(path)
    for name, (res, args) in SIGNATURES.items():
        fn = getattr(lib, name)
        fn.restype = res
        fn.argtypes = args
    _LIB = lib
    return lib


def _check(lib, st: int) -> int:
    if st < 0:
        msg = lib.gmmnlse_status_string(st).decode()
        if st == ECUDA:
            msg += ": " + lib.gmmnlse_last_cuda_error().decode()
        raise GmmnlseError(st, msg)
    return st


def _ptr(x) -> int:
    """Raw address of a torch tensor (device or host), a numpy array or an int."""
    if x is None:
        return 0
    if isinstance(x, int):
        return x
    if isinstance(x, np.ndarray):
        return x.ctypes.data
    return x.data_ptr()


class Plan:
    """Owner of one ``gmmnlse_plan``; methods mirror the C calls one to one."""

    def __init__(self, P, N, M, dt, dz, beta, S, f_R, h_R, omega0, n2, *, precision=0, shock=True,
                 tol=1e-6, max_iter=0, fixed_iter=0, contraction=0, raman=0, graph=0, stop_rule=0, async_call=0):
        self._lib = load_library()
        self._h = C.c_void_p()
        beta = np.ascontiguousarray(beta, dtype=np.float64).reshape(P, -1)
        general = isinstance(S, tuple)          # (S_K, S_R): the general form of Eq. 1
        if general:
            cplx = any(np.iscomplexobj(x) for x in S)
            SK, SR = (np.ascontiguousarray(x, dtype=np.complex128 if cplx else np.float64) for x in S)
            if SK.size != P ** 4 or SR.size != P ** 4:
                raise GmmnlseError(EINVAL, "S_K and S_R must hold P^4 entries each")
        else:
            S = np.ascontiguousarray(S, dtype=np.float64)
            if S.size != P ** 4:
                raise GmmnlseError(EINVAL, "S must hold P^4 entries")
        hR = None if h_R is None else np.ascontiguousarray(h_R, dtype=np.float64)
        if hR is not None and hR.size != N:
            raise GmmnlseError(EINVAL, "h_R must hold N samples")
        opt = Options(int(precision), int(bool(shock)), float(tol), int(max_iter), int(fixed_iter), int(contraction),
                      int(raman), int(graph), int(stop_rule), int(async_call))
        hp = None if hR is None else hR.ctypes.data_as(_DP)
        if general:
            st = self._lib.gmmnlse_plan_create_general(
                C.byref(self._h), P, N, M, dt, dz, beta.ctypes.data_as(_DP), beta.shape[1],
                C.cast(SK.ctypes.data, _DP), C.cast(SR.ctypes.data, _DP), int(cplx), f_R, hp, omega0, n2,
                C.byref(opt))
        else:
            st = self._lib.gmmnlse_plan_create(
                C.byref(self._h), P, N, M, dt, dz, beta.ctypes.data_as(_DP), beta.shape[1], S.ctypes.data_as(_DP),
                f_R, hp, omega0, n2, C.byref(opt))
        _check(self._lib, st)
        self.P, self.N, self.M, self.precision = P, N, M, int(precision)
        self.np_dtype = np.complex128 if precision else np.complex64

    # -- the three calls of the paper's problem statement ---------------------------------------
    def propagate(self, A_in, L, A_out, stream=None) -> int:
        """gmmnlse_propagate: device [P][N] in/out; returns OK or WARN_NOCONV."""
        return _check(self._lib, self._lib.gmmnlse_propagate(self._h, _ptr(A_in), float(L), _ptr(A_out),
                                                             _stream_ptr(stream)))

    def propagate_host(self, A_in: np.ndarray, L, A_out: np.ndarray) -> int:
        """gmmnlse_propagate_host: HOST numpy [P][N] buffers of the plan's precision."""
        for a in (A_in, A_out):
            if a.dtype != self.np_dtype or not a.flags.c_contiguous or a.size != self.P * self.N:
                raise GmmnlseError(EINVAL, "host buffers must be C-contiguous [P][N] of the plan's precision")
        return _check(self._lib, self._lib.gmmnlse_propagate_host(self._h, _ptr(A_in), float(L), _ptr(A_out)))

    def propagate_rk4ip(self, A_in, L, A_out, stream=None) -> int:
        """gmmnlse_propagate_rk4ip: the serial RK4IP integrator (step dz) on the same kernels."""
        return _check(self._lib, self._lib.gmmnlse_propagate_rk4ip(self._h, _ptr(A_in), float(L), _ptr(A_out),
                                                                   _stream_ptr(stream)))

    def nonlinear_op(self, A, dA) -> int:
        return _check(self._lib, self._lib.gmmnlse_nonlinear_op(self._h, _ptr(A), _ptr(dA)))

    # -- plane-axis sharding (one large step in pieces; the collectives are the caller's: sharded.py) -----
    def shard_begin(self, A_in) -> None:
        _check(self._lib, self._lib.gmmnlse_shard_begin(self._h, _ptr(A_in)))

    def shard_iterate(self, j_lo, j_hi, Mc, first, block_sum) -> None:
        _check(self._lib, self._lib.gmmnlse_shard_iterate(self._h, int(j_lo), int(j_hi), int(Mc), int(bool(first)),
                                                          _ptr(block_sum)))

    def shard_update(self, j_lo, j_hi, Mc, first, all_sums, shard, n_shards) -> float:
        err = C.c_double()
        _check(self._lib, self._lib.gmmnlse_shard_update(self._h, int(j_lo), int(j_hi), int(Mc), int(bool(first)),
                                                         _ptr(all_sums), int(shard), int(n_shards), C.byref(err)))
        return err.value

    def shard_advance(self, Mc, all_sums, n_shards) -> None:
        _check(self._lib, self._lib.gmmnlse_shard_advance(self._h, int(Mc), _ptr(all_sums), int(n_shards)))

    def shard_end(self, A_out) -> None:
        _check(self._lib, self._lib.gmmnlse_shard_end(self._h, _ptr(A_out)))

    def set_gain(self, g) -> None:
        """gmmnlse_set_gain: g[P] field gain in 1/m (None clears it)."""
        if g is None:
            _check(self._lib, self._lib.gmmnlse_set_gain(self._h, None))
            return
        g = np.ascontiguousarray(g, dtype=np.float64)
        if g.size != self.P:
            raise GmmnlseError(EINVAL, "gain must hold P entries")
        _check(self._lib, self._lib.gmmnlse_set_gain(self._h, g.ctypes.data_as(_DP)))

    def set_coupling(self, Q) -> None:
        """gmmnlse_set_coupling: Q[n][p] = Q_np complex [P][P] in 1/m (None clears it)."""
        if Q is None:
            _check(self._lib, self._lib.gmmnlse_set_coupling(self._h, None))
            return
        Q = np.ascontiguousarray(Q, dtype=np.complex128)
        if Q.size != self.P * self.P:
            raise GmmnlseError(EINVAL, "Q must hold P x P entries")
        _check(self._lib, self._lib.gmmnlse_set_coupling(self._h, C.cast(Q.ctypes.data, _DP)))

    def set_coupling_profile(self, f) -> None:
        """gmmnlse_set_coupling_profile: f(k dz / 2), k = 0..n-1, from the start of each call (None: constant)."""
        if f is None:
            _check(self._lib, self._lib.gmmnlse_set_coupling_profile(self._h, None, 0))
            return
        f = np.ascontiguousarray(f, dtype=np.float64)
        _check(self._lib, self._lib.gmmnlse_set_coupling_profile(self._h, f.ctypes.data_as(_DP), int(f.size)))

    def set_gain_saturation(self, g_sat: float) -> None:
        """gmmnlse_set_gain_saturation: g0 / I_sat in m/J (0 = off)."""
        _check(self._lib, self._lib.gmmnlse_set_gain_saturation(self._h, float(g_sat)))

    # -- helpers -----------------------------------------------------------------------------------
    def set_stream(self, stream) -> None:
        _check(self._lib, self._lib.gmmnlse_set_stream(self._h, _stream_ptr(stream)))

    def stats(self) -> dict:
        a, b, d = C.c_longlong(), C.c_longlong(), C.c_longlong()
        e = C.c_double()
        _check(self._lib, self._lib.gmmnlse_get_stats(self._h, C.byref(a), C.byref(b), C.byref(e), C.byref(d)))
        return dict(large_steps=a.value, iterations=b.value, last_err=e.value, not_converged=d.value)

    def launch_count(self) -> int:
        return int(self._lib.gmmnlse_launch_count(self._h))

    def profile_enable(self, on: bool = True) -> None:
        _check(self._lib, self._lib.gmmnlse_profile_enable(self._h, int(on)))

    def profile_get(self) -> dict:
        """{kind name: (total_ms, launches)} accumulated since profile_enable(True)."""
        out = {}
        for k, name in enumerate(KINDS):
            ms, n = C.c_double(), C.c_longlong()
            _check(self._lib, self._lib.gmmnlse_profile_get(self._h, k, C.byref(ms), C.byref(n)))
            out[name] = (ms.value, n.value)
        return out

    def debug_get_planes(self) -> np.ndarray:
        out = np.empty((self.M + 1, self.P, self.N), dtype=self.np_dtype)
        _check(self._lib, self._lib.gmmnlse_debug_get_planes(self._h, _ptr(out)))
        return out

    def debug_fft(self, x, out, rows: int, direction: int) -> None:
        _check(self._lib, self._lib.gmmnlse_debug_fft(self._h, _ptr(x), _ptr(out), rows, direction))

    def debug_pairs(self, A, V, n_planes: int) -> None:
        _check(self._lib, self._lib.gmmnlse_debug_pairs(self._h, _ptr(A), _ptr(V), n_planes))

    def debug_contract(self, V, U, n_planes: int) -> None:
        _check(self._lib, self._lib.gmmnlse_debug_contract(self._h, _ptr(V), _ptr(U), n_planes))

    def contraction_kind(self) -> int:
        """1 CUDA cores, 3 tcgen05 3xTF32, 7 tcgen05 kind::f16, 6 / 8 the low-rank pairs of those."""
        return int(self._lib.gmmnlse_contraction_kind(self._h))

    def lowrank_rank(self) -> int:
        return int(self._lib.gmmnlse_lowrank_rank(self._h))

    def sparse_info(self) -> dict:
        """contraction 9: {classes, work_fraction} of the block-sparse form (0 and 1.0 otherwise)."""
        c, f = C.c_int(), C.c_double()
        _check(self._lib, self._lib.gmmnlse_sparse_info(self._h, C.byref(c), C.byref(f)))
        return dict(classes=c.value, work_fraction=f.value)

    def loop_kind(self) -> int:
        return int(self._lib.gmmnlse_loop_kind(self._h))

    def raman_kind(self) -> int:
        """0 = no Raman term, 1 = FFT convolution, 2 = recursive (damped-oscillator) form."""
        return int(self._lib.gmmnlse_raman_kind(self._h))

    def debug_set_tc_chunk(self, k: int) -> None:
        _check(self._lib, self._lib.gmmnlse_debug_set_tc_chunk(self._h, int(k)))

    def destroy(self) -> None:
        if self._h:
            self._lib.gmmnlse_plan_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()


def overlap_tensor(F, dA: float) -> np.ndarray:
    """gmmnlse_overlap_tensor: S_plmn of Eq. 2 from P mode fields F[P][...grid] (any grid shape), on the GPU."""
    lib = load_library()
    F = np.ascontiguousarray(F, dtype=np.float64)
    P = F.shape[0]
    F = F.reshape(P, -1)
    S = np.empty((P, P, P, P), dtype=np.float64)
    _check(lib, lib.gmmnlse_overlap_tensor(P, F.shape[1], F.ctypes.data_as(_DP), float(dA), S.ctypes.data_as(_DP)))
    return S


def overlap_tensor_noalloc(F_dev, dA: float, S_dev, stream=None) -> None:
    """gmmnlse_overlap_tensor_noalloc: DEVICE fp64 tensors F_dev [P][G...] in, S_dev [P][P][P][P] out; allocates
    nothing, enqueues on `stream`, shares one static scratch array per device (calls must not overlap on the GPU)."""
    lib = load_library()
    P = int(F_dev.shape[0])
    G = int(F_dev.numel() // P)
    st = lib.gmmnlse_overlap_tensor_noalloc(P, G, _ptr(F_dev), float(dA), _ptr(S_dev), _stream_ptr(stream))
    if st == EUNSUPPORTED:
        raise GmmnlseError(st, lib.gmmnlse_last_cuda_error().decode())
    _check(lib, st)


def overlap_tensor_noalloc_limits() -> dict:
    lib = load_library()
    p, g, b = C.c_int(), C.c_longlong(), C.c_longlong()
    _check(lib, lib.gmmnlse_overlap_tensor_noalloc_limits(C.byref(p), C.byref(g), C.byref(b)))
    return dict(P_max=p.value, G_max=g.value, scratch_bytes=b.value)


def _stream_ptr(stream) -> int:
    if stream is None:
        return 0
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream          # torch.cuda.Stream


def plan_from_workload(w, **overrides) -> Plan:
    """Plan for a :class:`workloads.Workload` (its precision, shock, tol, M)."""
    kw = dict(precision=w.precision, shock=w.shock, tol=w.tol)
    kw.update(overrides)
    M = kw.pop("M", w.M)
    return Plan(w.P, w.N, M, w.dt, w.dz, w.beta, w.S, w.f_R, w.h_R, w.omega0, w.n2, **kw)
