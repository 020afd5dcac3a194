"""Thin ctypes binding of liblrp (include/lrp.h): argument marshalling only -- every step of the hot path
runs in the CUDA kernels behind the C ABI.  PyTorch is used for device memory and streams.

Layout convention of this binding: a "tall" n x k matrix (column-major, ld = n, as the C ABI wants) is a
contiguous CUDA float64 tensor of shape (k, n): element (i, c) lives at t[c, i].  `tall_from_numpy` /
`tall_to_numpy` convert from/to ordinary (n, k) numpy arrays.

There is no CPU fallback: if liblrp.so is missing (run `python -m paper_2607_06021_b200.build`) or no CUDA
device is present, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liblrp.so")

LRP_OK, LRP_ERR_BADARG, LRP_ERR_UNSUPPORTED_N, LRP_ERR_WORKSPACE, LRP_ERR_CUDA, LRP_WARN_NOCONV = 0, -1, -2, -3, -4, 1
LRP_ERR_STATIC_LIMIT = -5
TOPK_STATIC_MAX_N, TOPK_STATIC_MAX_NUM = 4194304, 256
MAX_SWEEPS_INFO = 32
LRP_FLAG_NO_QR_REUSE, LRP_FLAG_NO_NESTED_RHO, LRP_FLAG_NO_FUSED_RHO, LRP_FLAG_NO_CHOLQR_LEVERAGE = 1, 2, 4, 8
LRP_FLAG_NO_PRIORITY_STREAMS = 16
LRP_G_POISSON, LRP_G_HILBERT, LRP_G_KMATRIX = 0, 1, 2
SELECTIONS = {"topk": 0, "bernoulli": 1, "qdeim": 2, "deim": 3}
MATRIX_KINDS = {"hilbert": LRP_G_HILBERT, "kmatrix": LRP_G_KMATRIX}

EXPORTS = ["lrp_create", "lrp_destroy", "lrp_strerror", "lrp_last_cuda_error", "lrp_launch_count",
           "lrp_workspace_bytes", "lrp_dst1_workspace_bytes", "lrp_leverage_workspace_bytes",
           "lrp_scross_workspace_bytes", "lrp_set_workspace", "lrp_dst1_batched", "lrp_sample_fibers",
           "lrp_leverage_select", "lrp_scross", "lrp_cross_deim_solve", "lrp_lowrank_entries",
           "lrp_profile_enable", "lrp_profile_reset", "lrp_profile_count", "lrp_profile_get",
           "lrp_profile_timeline", "lrp_fp64_peak", "lrp_matrix_workspace_bytes", "lrp_cross_deim_matrix",
           "lrp_sample_matrix", "lrp_dense_workspace_bytes", "lrp_dense_poisson", "lrp_topk_static",
           "lrp_solve_host_workspace_bytes", "lrp_cross_deim_solve_host",
           "lrp_solve_batch_workspace_bytes", "lrp_cross_deim_solve_batch"]


class SolveOpts(C.Structure):
    _fields_ = [("tol", C.c_double), ("max_rank", C.c_int32), ("oversample", C.c_int32), ("max_sweeps", C.c_int32),
                ("tol_mode", C.c_int32), ("h_safeguard", C.c_void_p), ("n_safeguard", C.c_int32),
                ("d_U0", C.c_void_p), ("d_V0", C.c_void_p), ("ld0", C.c_int64), ("r0", C.c_int32),
                ("replay_sweeps", C.c_int32), ("h_replay_nI", C.c_void_p), ("h_replay_nJ", C.c_void_p),
                ("h_replay_I", C.c_void_p), ("h_replay_J", C.c_void_p), ("h_replay_keepI", C.c_void_p),
                ("h_replay_keepJ", C.c_void_p), ("replay_final_rank", C.c_int32), ("flags", C.c_int32),
                ("selection", C.c_int32), ("ls_seed", C.c_uint64), ("ls_c", C.c_double)]


class SolveInfo(C.Structure):
    _fields_ = [("rank", C.c_int32), ("sweeps", C.c_int32), ("converged", C.c_int32),
                ("rho", C.c_double), ("indicator", C.c_double), ("eta1", C.c_double), ("eta2", C.c_double),
                ("snorm", C.c_double), ("smin_full", C.c_double),
                ("nI", C.c_int32 * MAX_SWEEPS_INFO), ("nJ", C.c_int32 * MAX_SWEEPS_INFO),
                ("rank_per_sweep", C.c_int32 * MAX_SWEEPS_INFO),
                ("rho_per_sweep", C.c_double * MAX_SWEEPS_INFO), ("ind_per_sweep", C.c_double * MAX_SWEEPS_INFO),
                ("ms_dst_fwd", C.c_float), ("ms_select", C.c_float), ("ms_sample", C.c_float), ("ms_qr", C.c_float),
                ("ms_core", C.c_float), ("ms_rebuild", C.c_float), ("ms_stop", C.c_float), ("ms_dst_inv", C.c_float),
                ("ms_total", C.c_float), ("launches", C.c_int64)]


_lib = None


def load_library():
    """Load liblrp.so and declare the prototypes; raises if the library is not built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2607_06021_b200.build` "
                           "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, i32, i64, dbl, sz = C.c_void_p, C.c_int32, C.c_int64, C.c_double, C.c_size_t
    lib.lrp_create.argtypes = [C.POINTER(vp), C.c_int, vp]; lib.lrp_create.restype = C.c_int
    lib.lrp_destroy.argtypes = [vp]; lib.lrp_destroy.restype = C.c_int
    lib.lrp_strerror.argtypes = [C.c_int]; lib.lrp_strerror.restype = C.c_char_p
    lib.lrp_last_cuda_error.argtypes = [vp]; lib.lrp_last_cuda_error.restype = C.c_int
    lib.lrp_launch_count.argtypes = [vp]; lib.lrp_launch_count.restype = i64
    lib.lrp_workspace_bytes.argtypes = [i64, i32, i32, i32]; lib.lrp_workspace_bytes.restype = sz
    lib.lrp_dst1_workspace_bytes.argtypes = [i64, i32]; lib.lrp_dst1_workspace_bytes.restype = sz
    lib.lrp_leverage_workspace_bytes.argtypes = [i64, i32]; lib.lrp_leverage_workspace_bytes.restype = sz
    lib.lrp_scross_workspace_bytes.argtypes = [i64, i32, i32]; lib.lrp_scross_workspace_bytes.restype = sz
    lib.lrp_set_workspace.argtypes = [vp, vp, sz]; lib.lrp_set_workspace.restype = C.c_int
    lib.lrp_dst1_batched.argtypes = [vp, i64, i32, vp, i64, vp, i64, dbl]; lib.lrp_dst1_batched.restype = C.c_int
    lib.lrp_sample_fibers.argtypes = [vp, i64, i32, vp, i64, vp, vp, i64, vp, i32, vp, i32, vp, i64, vp, i64]
    lib.lrp_sample_fibers.restype = C.c_int
    lib.lrp_leverage_select.argtypes = [vp, i64, i32, vp, i64, i32, C.c_int, vp, vp]; lib.lrp_leverage_select.restype = C.c_int
    lib.lrp_scross.argtypes = [vp, i64, vp, i64, i32, vp, i64, i32, vp, vp, vp, i64, vp, vp, i64, vp, vp,
                               C.POINTER(i32), C.POINTER(dbl)]
    lib.lrp_scross.restype = C.c_int
    lib.lrp_cross_deim_solve.argtypes = [vp, i64, i32, vp, i64, vp, vp, i64, C.POINTER(SolveOpts), vp, i64, vp, vp, i64,
                                         C.POINTER(SolveInfo), vp, vp, vp, vp, vp, vp, vp, i64]
    lib.lrp_cross_deim_solve.restype = C.c_int
    lib.lrp_solve_host_workspace_bytes.argtypes = [i64, i32, i32, i32, i32]; lib.lrp_solve_host_workspace_bytes.restype = sz
    lib.lrp_cross_deim_solve_host.argtypes = [vp, i64, i32, i32, vp, i64, vp, vp, i64, vp, vp, i64, vp, vp, i64, vp]
    lib.lrp_cross_deim_solve_host.restype = C.c_int
    lib.lrp_solve_batch_workspace_bytes.argtypes = [i64, i32, i32, i32, i32]; lib.lrp_solve_batch_workspace_bytes.restype = sz
    lib.lrp_cross_deim_solve_batch.argtypes = [vp, i64, i32, i32, vp, i64, vp, vp, i64, vp, vp, i64, vp, vp, i64, vp]
    lib.lrp_cross_deim_solve_batch.restype = C.c_int
    lib.lrp_matrix_workspace_bytes.argtypes = [i64, i32, i32, i32]; lib.lrp_matrix_workspace_bytes.restype = sz
    lib.lrp_cross_deim_matrix.argtypes = [vp, i32, i64, C.POINTER(SolveOpts), vp, i64, vp, vp, i64, C.POINTER(SolveInfo),
                                          vp, vp, vp, vp, vp, vp, vp, i64]
    lib.lrp_cross_deim_matrix.restype = C.c_int
    lib.lrp_sample_matrix.argtypes = [vp, i32, i64, vp, i32, vp, i32, vp, i64, vp, i64]; lib.lrp_sample_matrix.restype = C.c_int
    lib.lrp_dense_workspace_bytes.argtypes = [i64]; lib.lrp_dense_workspace_bytes.restype = sz
    lib.lrp_dense_poisson.argtypes = [vp, i64, vp, i64, vp, i64]; lib.lrp_dense_poisson.restype = C.c_int
    lib.lrp_lowrank_entries.argtypes = [vp, i64, i32, vp, i64, vp, vp, i64, vp, vp, i64, vp]
    lib.lrp_lowrank_entries.restype = C.c_int
    lib.lrp_topk_static.argtypes = [vp, i64, vp, i32, vp]; lib.lrp_topk_static.restype = C.c_int
    lib.lrp_profile_enable.argtypes = [vp, C.c_int]; lib.lrp_profile_enable.restype = C.c_int
    lib.lrp_profile_timeline.argtypes = [vp, C.c_char_p]; lib.lrp_profile_timeline.restype = C.c_int
    lib.lrp_profile_reset.argtypes = [vp]; lib.lrp_profile_reset.restype = C.c_int
    lib.lrp_fp64_peak.argtypes = [vp, C.POINTER(dbl), C.POINTER(dbl)]; lib.lrp_fp64_peak.restype = C.c_int
    lib.lrp_profile_count.argtypes = []; lib.lrp_profile_count.restype = C.c_int
    lib.lrp_profile_get.argtypes = [vp, C.c_int, C.POINTER(C.c_char_p), C.POINTER(i64), C.POINTER(dbl),
                                    C.POINTER(dbl), C.POINTER(dbl)]
    lib.lrp_profile_get.restype = C.c_int
    _lib = lib
    return lib


class LrpError(RuntimeError):
    def __init__(self, code, where, cuda=0):
        msg = load_library().lrp_strerror(code).decode()
        super().__init__(f"{where}: {msg} (code {code}, cudaError {cuda})")
        self.code = code


def _torch():
    import torch
    return torch


def tall_from_numpy(a: np.ndarray, device="cuda:0"):
    """(n, k) numpy -> device tall tensor of shape (k, n)."""
    torch = _torch()
    a = np.asarray(a, dtype=np.float64)
    if a.ndim == 1:
        a = a[:, None]
    return torch.from_numpy(np.ascontiguousarray(a.T)).to(device)


def tall_to_numpy(t) -> np.ndarray:
    return t.detach().cpu().numpy().T.copy()


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else C.c_void_p(0)


def _check_tall(t, name):
    torch = _torch()
    if not (t.is_cuda and t.dtype == torch.float64 and t.dim() == 2 and (t.stride(1) == 1 or t.shape[1] == 1)):
        raise ValueError(f"{name}: expected a CUDA float64 tensor of shape (cols, n) with contiguous rows")
    ld = t.stride(0) if t.shape[0] > 1 else t.shape[1]
    return t.shape[0], t.shape[1], max(ld, t.shape[1])


def topk_static(scores, num_select: int, out, stream=None):
    """lrp_topk_static (include/lrp.h): allocation-free top-k into the caller's `out` (int32, >= num_select elements) on
    `stream` (a torch.cuda.Stream, default: the current one).  n <= TOPK_STATIC_MAX_N, num_select <= TOPK_STATIC_MAX_NUM.
    The library keeps one built-in scratch array per GPU: overlapping calls race."""
    torch = _torch()
    if not (scores.is_cuda and scores.dtype == torch.float64 and scores.dim() == 1 and scores.is_contiguous()):
        raise ValueError("scores: contiguous 1-D float64 CUDA tensor")
    if not (out.is_cuda and out.dtype == torch.int32 and out.is_contiguous() and out.numel() >= num_select):
        raise ValueError("out: contiguous int32 CUDA tensor with room for num_select indices")
    st = stream if stream is not None else torch.cuda.current_stream(scores.device)
    with torch.cuda.device(scores.device):
        rc = load_library().lrp_topk_static(C.c_void_p(st.cuda_stream), scores.numel(), _ptr(scores), int(num_select), _ptr(out))
    if rc < 0:
        raise LrpError(rc, "lrp_topk_static")
    return out[:num_select]


class Context:
    """Owns an lrp_ctx bound to a device and to torch's current stream on it, plus the workspace tensor."""

    def __init__(self, device: int = 0, stream=None):
        torch = _torch()
        self.lib = load_library()
        if not torch.cuda.is_available():
            raise RuntimeError("liblrp needs a CUDA device (no CPU fallback)")
        self.device = torch.device("cuda", device)
        torch.cuda.set_device(self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        h = C.c_void_p()
        rc = self.lib.lrp_create(C.byref(h), device, C.c_void_p(self.stream.cuda_stream))
        if rc != 0:
            raise LrpError(rc, "lrp_create")
        self.h = h
        self._ws = None

    def close(self):
        if getattr(self, "h", None):
            self.lib.lrp_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc, where):
        if rc < 0:
            raise LrpError(rc, where, self.lib.lrp_last_cuda_error(self.h))
        return rc

    def launch_count(self) -> int:
        return int(self.lib.lrp_launch_count(self.h))

    def profile_enable(self, on):
        """on = True/1: per-kernel times with the library's streams serialised; on = 2: timeline mode (real overlap)."""
        self._check(self.lib.lrp_profile_enable(self.h, int(on)), "lrp_profile_enable")

    def profile_timeline(self, path: str):
        self._check(self.lib.lrp_profile_timeline(self.h, path.encode()), "lrp_profile_timeline")

    def fp64_peak(self) -> dict:
        """Measured fp64 throughput (TFLOP/s) of plain DFMA and of the fp64 tensor pipe (DMMA)."""
        a, b = C.c_double(), C.c_double()
        self._check(self.lib.lrp_fp64_peak(self.h, C.byref(a), C.byref(b)), "lrp_fp64_peak")
        return {"dfma_tflops": a.value, "dmma_tflops": b.value}

    def profile_reset(self):
        self._check(self.lib.lrp_profile_reset(self.h), "lrp_profile_reset")

    def profile(self) -> dict:
        """{kernel class: dict(count, ms, bytes, flops)} for the classes that launched since the last reset."""
        out = {}
        for i in range(self.lib.lrp_profile_count()):
            name, cnt = C.c_char_p(), C.c_int64()
            ms, by, fl = C.c_double(), C.c_double(), C.c_double()
            self._check(self.lib.lrp_profile_get(self.h, i, C.byref(name), C.byref(cnt), C.byref(ms), C.byref(by),
                                                 C.byref(fl)), "lrp_profile_get")
            if cnt.value:
                out[name.value.decode()] = dict(count=cnt.value, ms=ms.value, bytes=by.value, flops=fl.value)
        return out

    def ensure_workspace(self, nbytes: int, exact: bool = False):
        """Grow the workspace tensor to nbytes (exact: make it exactly nbytes -- lrp_cross_deim_solve_host reads the
        number of lanes off the workspace size)."""
        torch = _torch()
        if self._ws is None or self._ws.numel() < nbytes or (exact and self._ws.numel() != nbytes):
            self._ws = None
            self._ws = torch.empty(max(int(nbytes), 256), dtype=torch.uint8, device=self.device)
            self._check(self.lib.lrp_set_workspace(self.h, _ptr(self._ws), self._ws.numel()), "lrp_set_workspace")

    def release_workspace(self):
        """Drop the workspace tensor (the next call sizes a new one)."""
        self._check(self.lib.lrp_set_workspace(self.h, C.c_void_p(0), 0), "lrp_set_workspace")
        self._ws = None

    # ------------------------------------------------------------------ the five calls of the boundary
    def dst1_batched(self, x, out=None, scale: float = 1.0):
        """out(:, b) = scale * DST-I(x(:, b)); x, out tall tensors of shape (batch, n).  out may be x."""
        torch = _torch()
        batch, n, ld_in = _check_tall(x, "x")
        if out is None:
            out = torch.empty_like(x)
        _, _, ld_out = _check_tall(out, "out")
        self.ensure_workspace(self.lib.lrp_dst1_workspace_bytes(n, batch))
        self._check(self.lib.lrp_dst1_batched(self.h, n, batch, _ptr(x), ld_in, _ptr(out), ld_out, float(scale)),
                    "lrp_dst1_batched")
        return out

    def sample_fibers(self, Uh, S, Vh, I=None, J=None):
        """C = G(:, J) and Rt = G(I, :)^T as tall tensors (|J|, n), (|I|, n); I, J int32 CUDA tensors."""
        torch = _torch()
        r, n, ldu = _check_tall(Uh, "Uh")
        _, _, ldv = _check_tall(Vh, "Vh")
        Cm = torch.empty((J.numel(), n), dtype=torch.float64, device=Uh.device) if J is not None else None
        Rt = torch.empty((I.numel(), n), dtype=torch.float64, device=Uh.device) if I is not None else None
        self._check(self.lib.lrp_sample_fibers(self.h, n, r, _ptr(Uh), ldu, _ptr(S), _ptr(Vh), ldv,
                                               _ptr(I), I.numel() if I is not None else 0,
                                               _ptr(J), J.numel() if J is not None else 0,
                                               _ptr(Cm), n, _ptr(Rt), n), "lrp_sample_fibers")
        return Cm, Rt

    def leverage_select(self, A, num_select: int, assume_orthonormal: bool = False):
        torch = _torch()
        k, n, lda = _check_tall(A, "A")
        idx = torch.empty(max(num_select, 1), dtype=torch.int32, device=A.device)
        scores = torch.empty(n, dtype=torch.float64, device=A.device)
        self.ensure_workspace(self.lib.lrp_leverage_workspace_bytes(n, k))
        self._check(self.lib.lrp_leverage_select(self.h, n, k, _ptr(A), lda, num_select, int(assume_orthonormal),
                                                 _ptr(idx), _ptr(scores)), "lrp_leverage_select")
        return idx[:num_select], scores

    def scross(self, Cm, Rt, I, J):
        torch = _torch()
        k, n, ldc = _check_tall(Cm, "C")
        l, _, ldr = _check_tall(Rt, "Rt")
        p = min(k, l)
        U = torch.empty((p, n), dtype=torch.float64, device=Cm.device)
        V = torch.empty((p, n), dtype=torch.float64, device=Cm.device)
        S = torch.empty(p, dtype=torch.float64, device=Cm.device)
        rC = torch.empty(k, dtype=torch.float64, device=Cm.device)
        rR = torch.empty(l, dtype=torch.float64, device=Cm.device)
        rank = C.c_int32(0)
        smin = C.c_double(0.0)
        self.ensure_workspace(self.lib.lrp_scross_workspace_bytes(n, k, l))
        self._check(self.lib.lrp_scross(self.h, n, _ptr(Cm), ldc, k, _ptr(Rt), ldr, l, _ptr(I), _ptr(J),
                                        _ptr(U), n, _ptr(S), _ptr(V), n, _ptr(rC), _ptr(rR),
                                        C.byref(rank), C.byref(smin)), "lrp_scross")
        r = rank.value
        return dict(U=U[:r], S=S[:r], V=V[:r], S_full=S, rC=rC, rR=rR, rank=r, smin_full=smin.value)

    def _run_solve(self, n, dev, Kc, max_rank, call, *, tol, oversample, max_sweeps, safeguard, tol_mode, U0, V0, replay,
                   want_spectral, flags, selection="topk", ls_seed=0, ls_c=0.0):
        """Marshals lrp_solve_opts / lrp_solve_info / trace buffers and runs `call(opts, outputs...)`."""
        torch = _torch()
        # outputs: only the first info.rank columns are defined (and returned); no fill kernels on the solve's path
        UW = torch.empty((max_rank, n), dtype=torch.float64, device=dev)
        VW = torch.empty((max_rank, n), dtype=torch.float64, device=dev)
        SW = torch.empty(max_rank, dtype=torch.float64, device=dev)
        o = SolveOpts()
        o.tol, o.max_rank, o.oversample, o.max_sweeps, o.tol_mode = tol, max_rank, oversample, max_sweeps, tol_mode
        o.flags = int(flags)
        o.selection = SELECTIONS[selection] if isinstance(selection, str) else int(selection)
        o.ls_seed, o.ls_c = int(ls_seed), float(ls_c)
        keep = []
        if safeguard is not None:
            sg = np.ascontiguousarray(safeguard, dtype=np.int32); keep.append(sg)
            o.h_safeguard, o.n_safeguard = sg.ctypes.data, sg.size
        if U0 is not None:
            r0, _, ld0 = _check_tall(U0, "U0")
            o.d_U0, o.d_V0, o.ld0, o.r0 = U0.data_ptr(), V0.data_ptr(), ld0, r0
        if replay is not None:
            nI = np.array([len(s["I"]) for s in replay], dtype=np.int32)
            nJ = np.array([len(s["J"]) for s in replay], dtype=np.int32)
            Icat = np.ascontiguousarray(np.concatenate([np.asarray(s["I"], dtype=np.int32) for s in replay]))
            Jcat = np.ascontiguousarray(np.concatenate([np.asarray(s["J"], dtype=np.int32) for s in replay]))
            keep += [nI, nJ, Icat, Jcat]
            o.replay_sweeps = len(replay)
            o.h_replay_nI, o.h_replay_nJ, o.h_replay_I, o.h_replay_J = nI.ctypes.data, nJ.ctypes.data, Icat.ctypes.data, Jcat.ctypes.data
            if replay[0].get("keepI") is not None:
                kI = np.ascontiguousarray(np.concatenate([np.asarray(s["keepI"], dtype=np.uint8) for s in replay]))
                kJ = np.ascontiguousarray(np.concatenate([np.asarray(s["keepJ"], dtype=np.uint8) for s in replay]))
                keep += [kI, kJ]
                o.h_replay_keepI, o.h_replay_keepJ = kI.ctypes.data, kJ.ctypes.data
            o.replay_final_rank = int(replay[-1].get("final_rank") or 0)
        info = SolveInfo()
        trI = np.zeros(MAX_SWEEPS_INFO * Kc, dtype=np.int32); trJ = np.zeros_like(trI)
        tkI = np.zeros(MAX_SWEEPS_INFO * Kc, dtype=np.uint8); tkJ = np.zeros_like(tkI)
        Uhat = Vhat = Shat = None
        if want_spectral:
            Uhat = torch.empty((Kc, n), dtype=torch.float64, device=dev)
            Vhat = torch.empty((Kc, n), dtype=torch.float64, device=dev)
            Shat = torch.empty(Kc, dtype=torch.float64, device=dev)
        rc = call(o, UW, SW, VW, info, trI, trJ, tkI, tkJ, Uhat, Shat, Vhat)
        del keep
        sweeps, r = info.sweeps, info.rank
        trace, oi, oj = [], 0, 0
        for s in range(sweeps):
            a, b = info.nI[s], info.nJ[s]
            trace.append(dict(I=trI[oi:oi + a].copy(), J=trJ[oj:oj + b].copy(),
                              keepI=tkI[oi:oi + a].astype(bool), keepJ=tkJ[oj:oj + b].astype(bool),
                              rank=info.rank_per_sweep[s], rho=info.rho_per_sweep[s], ind=info.ind_per_sweep[s]))
            oi += a; oj += b
        res = dict(UW=UW[:r], SW=SW[:r], VW=VW[:r], rank=r, sweeps=sweeps, converged=bool(info.converged),
                   code=rc, trace=trace, info=info)
        if want_spectral:
            rk = info.rank_per_sweep[sweeps - 1]
            res.update(Uhat=Uhat[:rk], Shat=Shat[:rk], Vhat=Vhat[:rk])
        return res

    def cross_deim_solve(self, UF, SF, VF, *, tol, max_rank, oversample=8, max_sweeps=20, safeguard=None,
                         tol_mode=0, U0=None, V0=None, replay=None, want_spectral=False, flags=0, selection="topk", ls_seed=0,
                         ls_c=0.0):
        """Low-rank Poisson solve.  UF, VF: tall tensors (rF, n) in physical space, SF: (rF,) CUDA tensor.
        replay: list of dicts {I, J, keepI, keepJ} (numpy) + optional 'final_rank' on the last one."""
        rF, n, ldu = _check_tall(UF, "UF")
        _, _, ldv = _check_tall(VF, "VF")
        self.ensure_workspace(self.lib.lrp_workspace_bytes(n, rF, max_rank, oversample))

        def call(o, UW, SW, VW, info, trI, trJ, tkI, tkJ, Uhat, Shat, Vhat):
            return self._check(self.lib.lrp_cross_deim_solve(
                self.h, n, rF, _ptr(UF), ldu, _ptr(SF), _ptr(VF), ldv, C.byref(o), _ptr(UW), n, _ptr(SW), _ptr(VW), n,
                C.byref(info), trI.ctypes.data, trJ.ctypes.data, tkI.ctypes.data, tkJ.ctypes.data,
                _ptr(Uhat), _ptr(Shat), _ptr(Vhat), n), "lrp_cross_deim_solve")
        return self._run_solve(n, UF.device, 2 * (max_rank + oversample), max_rank, call, tol=tol, oversample=oversample,
                               max_sweeps=max_sweeps, safeguard=safeguard, tol_mode=tol_mode, U0=U0, V0=V0, replay=replay,
                               want_spectral=want_spectral, flags=flags, selection=selection, ls_seed=ls_seed, ls_c=ls_c)

    def cross_deim_solve_host(self, problems, outputs, *, tol, max_rank, oversample=8, max_sweeps=20, safeguard=None,
                              tol_mode=0, flags=0, selection="topk", ls_seed=0, ls_c=0.0, lanes=2):
        """lrp_cross_deim_solve_host: a batch of independent low-rank Poisson solves whose factors live in HOST memory.
        problems: list of (UF, SF, VF) CPU float64 tensors, UF / VF tall (rF, n) with contiguous rows, SF (rF,);
        outputs: list of (UW, SW, VW) CPU tensors of the same length, UW / VW (max_rank, n), SW (max_rank,) -- entries may
        repeat (a pool of >= 2 buffers) when earlier results are no longer needed.  Pinned tensors let the copies of the
        neighbouring problems overlap the solve; pageable ones work without overlap.  Returns one dict per problem
        (rank, sweeps, converged, info); the leading `rank` rows of its output tensors hold the factors.  lanes: 1 or 2
        solves in flight (sizes the workspace; include/lrp.h); outputs may repeat only between problems an even distance apart."""
        torch = _torch()

        def chk(t, name, rows=None):
            if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
                raise ValueError(f"{name}: expected a contiguous CPU float64 tensor")
            if rows is not None and (t.dim() != 2 or t.shape[0] != rows[0] or t.shape[1] != rows[1]):
                raise ValueError(f"{name}: expected shape {rows}")
        if len(problems) != len(outputs):
            raise ValueError("problems and outputs must have the same length")
        if not problems:
            return []
        rF, n = problems[0][0].shape
        for UF, SF, VF in problems:
            chk(UF, "UF", (rF, n)); chk(VF, "VF", (rF, n)); chk(SF, "SF")
            if SF.numel() != rF:
                raise ValueError("SF: expected rF values")
        for UW, SW, VW in outputs:
            chk(UW, "UW", (max_rank, n)); chk(VW, "VW", (max_rank, n)); chk(SW, "SW")
            if SW.numel() < max_rank:
                raise ValueError("SW: expected max_rank values of room")
        need = self.lib.lrp_solve_host_workspace_bytes(n, rF, max_rank, oversample, int(lanes))
        if need == 0:
            raise LrpError(-1, "lrp_solve_host_workspace_bytes (unsupported n, rank cap or lane count)")
        self.ensure_workspace(need, exact=True)
        o = SolveOpts()
        o.tol, o.max_rank, o.oversample, o.max_sweeps, o.tol_mode = tol, max_rank, oversample, max_sweeps, tol_mode
        o.flags = int(flags)
        o.selection = SELECTIONS[selection] if isinstance(selection, str) else int(selection)
        o.ls_seed, o.ls_c = int(ls_seed), float(ls_c)
        sg = None
        if safeguard is not None:
            sg = np.ascontiguousarray(safeguard, dtype=np.int32)
            o.h_safeguard, o.n_safeguard = sg.ctypes.data, sg.size
        P = len(problems)
        arr = lambda ts: (C.c_void_p * P)(*[t.data_ptr() for t in ts])
        hUF, hSF, hVF = arr([p[0] for p in problems]), arr([p[1] for p in problems]), arr([p[2] for p in problems])
        hUW, hSW, hVW = arr([q[0] for q in outputs]), arr([q[1] for q in outputs]), arr([q[2] for q in outputs])
        infos = (SolveInfo * P)()
        rc = self._check(self.lib.lrp_cross_deim_solve_host(self.h, n, rF, P, hUF, n, hSF, hVF, n, C.byref(o),
                                                            hUW, n, hSW, hVW, n, infos), "lrp_cross_deim_solve_host")
        del sg
        return [dict(rank=infos[p].rank, sweeps=infos[p].sweeps, converged=bool(infos[p].converged), code=rc, info=infos[p])
                for p in range(P)]

    def cross_deim_solve_batch(self, problems, *, tol, max_rank, oversample=8, max_sweeps=20, safeguard=None,
                               tol_mode=0, flags=0, selection="topk", ls_seed=0, ls_c=0.0, lanes=2, outputs=None):
        """lrp_cross_deim_solve_batch: independent problems with DEVICE factors, two solves in flight when lanes = 2.
        problems: list of (UF, SF, VF) CUDA tensors as for cross_deim_solve.  Returns one dict per problem like
        cross_deim_solve (UW, SW, VW, rank, sweeps, converged, info).  outputs: optional list of preallocated
        (UW (max_rank, n), SW (max_rank,), VW (max_rank, n)) CUDA tensors, one distinct triple per problem."""
        torch = _torch()
        if not problems:
            return []
        rF, n, ldu = _check_tall(problems[0][0], "UF")
        _, _, ldv = _check_tall(problems[0][2], "VF")
        for UF, SF, VF in problems:
            if _check_tall(UF, "UF") != (rF, n, ldu) or _check_tall(VF, "VF") != (rF, n, ldv):
                raise ValueError("all problems must share n, rF and the leading dimensions")
        need = self.lib.lrp_solve_batch_workspace_bytes(n, rF, max_rank, oversample, int(lanes))
        if need == 0:
            raise LrpError(-1, "lrp_solve_batch_workspace_bytes (unsupported n, rank cap or lane count)")
        self.ensure_workspace(need, exact=True)
        o = SolveOpts()
        o.tol, o.max_rank, o.oversample, o.max_sweeps, o.tol_mode = tol, max_rank, oversample, max_sweeps, tol_mode
        o.flags = int(flags)
        o.selection = SELECTIONS[selection] if isinstance(selection, str) else int(selection)
        o.ls_seed, o.ls_c = int(ls_seed), float(ls_c)
        sg = None
        if safeguard is not None:
            sg = np.ascontiguousarray(safeguard, dtype=np.int32)
            o.h_safeguard, o.n_safeguard = sg.ctypes.data, sg.size
        P = len(problems)
        dev = problems[0][0].device
        outs = outputs if outputs is not None else [
            (torch.empty((max_rank, n), dtype=torch.float64, device=dev), torch.empty(max_rank, dtype=torch.float64, device=dev),
             torch.empty((max_rank, n), dtype=torch.float64, device=dev)) for _ in range(P)]
        if len(outs) != P or any(q[0].shape != (max_rank, n) or q[2].shape != (max_rank, n) or q[1].numel() < max_rank for q in outs):
            raise ValueError("outputs: one (UW (max_rank, n), SW (max_rank,), VW (max_rank, n)) triple per problem")
        arr = lambda ts: (C.c_void_p * P)(*[t.data_ptr() for t in ts])
        infos = (SolveInfo * P)()
        rc = self._check(self.lib.lrp_cross_deim_solve_batch(
            self.h, n, rF, P, arr([p[0] for p in problems]), ldu, arr([p[1] for p in problems]), arr([p[2] for p in problems]), ldv,
            C.byref(o), arr([q[0] for q in outs]), n, arr([q[1] for q in outs]), arr([q[2] for q in outs]), n, infos),
            "lrp_cross_deim_solve_batch")
        del sg
        return [dict(UW=outs[p][0][:infos[p].rank], SW=outs[p][1][:infos[p].rank], VW=outs[p][2][:infos[p].rank], rank=infos[p].rank,
                     sweeps=infos[p].sweeps, converged=bool(infos[p].converged), code=rc, info=infos[p]) for p in range(P)]

    def cross_deim_matrix(self, kind, n, U0, V0, *, tol, max_rank, oversample=8, max_sweeps=20, safeguard=None,
                          tol_mode=0, replay=None, want_spectral=False, flags=0, selection="topk", ls_seed=0, ls_c=0.0):
        """Cross-DEIM on a closed-form test matrix of eq. (6) (kind 'hilbert' or 'kmatrix', n x n).  U0, V0: tall tensors
        (r0, n), the initial guess of Alg. 4.  Returns the same dictionary as cross_deim_solve (UW, SW, VW = the factors)."""
        k = MATRIX_KINDS[kind] if isinstance(kind, str) else int(kind)
        r0, n0, _ = _check_tall(U0, "U0")
        if n0 != n:
            raise ValueError("U0 must have n rows")
        self.ensure_workspace(self.lib.lrp_matrix_workspace_bytes(n, r0, max_rank, oversample))

        def call(o, UW, SW, VW, info, trI, trJ, tkI, tkJ, Uhat, Shat, Vhat):
            return self._check(self.lib.lrp_cross_deim_matrix(
                self.h, k, n, C.byref(o), _ptr(UW), n, _ptr(SW), _ptr(VW), n, C.byref(info),
                trI.ctypes.data, trJ.ctypes.data, tkI.ctypes.data, tkJ.ctypes.data,
                _ptr(Uhat), _ptr(Shat), _ptr(Vhat), n), "lrp_cross_deim_matrix")
        return self._run_solve(n, U0.device, 2 * (max_rank + oversample), max_rank, call, tol=tol, oversample=oversample,
                               max_sweeps=max_sweeps, safeguard=safeguard, tol_mode=tol_mode, U0=U0, V0=V0, replay=replay,
                               want_spectral=want_spectral, flags=flags, selection=selection, ls_seed=ls_seed, ls_c=ls_c)

    def sample_matrix(self, kind, n, I=None, J=None):
        """Fibers of a test matrix: C = G(:, J) as (|J|, n), Rt = G(I, :)^T as (|I|, n)."""
        torch = _torch()
        k = MATRIX_KINDS[kind] if isinstance(kind, str) else int(kind)
        Cm = torch.empty((J.numel(), n), dtype=torch.float64, device=self.device) if J is not None else None
        Rt = torch.empty((I.numel(), n), dtype=torch.float64, device=self.device) if I is not None else None
        self._check(self.lib.lrp_sample_matrix(self.h, k, n, _ptr(I), I.numel() if I is not None else 0,
                                               _ptr(J), J.numel() if J is not None else 0, _ptr(Cm), n, _ptr(Rt), n),
                    "lrp_sample_matrix")
        return Cm, Rt

    def dense_poisson(self, F):
        """Full-rank DST solve of section 3.1 for a dense right-hand side: F a CUDA float64 tensor whose element (i, j) is at
        F[j, i] (column-major n x n, like every tall tensor here); returns W in the same layout."""
        torch = _torch()
        n = F.shape[0]
        Wd = torch.empty_like(F)
        self.ensure_workspace(self.lib.lrp_dense_workspace_bytes(n))
        self._check(self.lib.lrp_dense_poisson(self.h, n, _ptr(F), n, _ptr(Wd), n), "lrp_dense_poisson")
        return Wd

    def lowrank_entries(self, U, S, V, rows, cols):
        torch = _torch()
        r, n, ldu = _check_tall(U, "U")
        _, _, ldv = _check_tall(V, "V")
        out = torch.empty(rows.numel(), dtype=torch.float64, device=U.device)
        self._check(self.lib.lrp_lowrank_entries(self.h, n, r, _ptr(U), ldu, _ptr(S), _ptr(V), ldv,
                                                 _ptr(rows), _ptr(cols), rows.numel(), _ptr(out)), "lrp_lowrank_entries")
        return out
