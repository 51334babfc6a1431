"""Thin ctypes binding of include/epo.h -- same names, argument marshalling only.

Every step of the path runs in the CUDA kernels of libepo.so; there is no Python or CPU fallback: if
the library is missing (not built) importing this module raises, and without a CUDA device
`epo_create` fails with EPO_ERR_CUDA.  Arrays may be numpy arrays (host pointers) or torch tensors
(host or CUDA); the library detects which.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libepo.so")

EPO_OK, EPO_ERR_INVALID_ARG, EPO_ERR_BAD_STATE, EPO_ERR_OUT_OF_MEMORY, EPO_ERR_CUDA, EPO_ERR_UNSUPPORTED = range(6)
_STATUS = {0: "EPO_OK", 1: "EPO_ERR_INVALID_ARG", 2: "EPO_ERR_BAD_STATE", 3: "EPO_ERR_OUT_OF_MEMORY",
           4: "EPO_ERR_CUDA", 5: "EPO_ERR_UNSUPPORTED"}

# every symbol include/epo.h declares (tests check that the library exports exactly these)
SYMBOLS = ["epo_config_default", "epo_create", "epo_destroy", "epo_extract_edges", "epo_extract_edges_rgb", "epo_set_views", "epo_build_viewgraph", "epo_set_pairs", "epo_loss_grad", "epo_loss_grad_joint", "epo_get_joint_variables",
           "epo_step", "epo_get_poses", "epo_get_poses_f64", "epo_reset", "epo_get_edge_counts", "epo_get_edge_list",
           "epo_get_dtf", "epo_get_pair_order", "epo_get_trace", "epo_get_work", "epo_get_pair_subset", "epo_time_loss_grad_kernel", "epo_time_gather_ceiling",
           "epo_edt_no_alloc", "epo_get_state_size", "epo_get_state", "epo_set_state", "epo_last_error", "epo_version"]


class EpoConfig(C.Structure):
    _fields_ = [("n_views", C.c_int32), ("width", C.c_int32), ("height", C.c_int32), ("huber_delta", C.c_float),
                ("clamp_start", C.c_float), ("clamp_end", C.c_float), ("clamp_steps", C.c_int32),
                ("lr_max", C.c_float), ("warmup_steps", C.c_int32), ("max_steps", C.c_int32),
                ("beta1", C.c_float), ("beta2", C.c_float), ("adam_eps", C.c_float), ("eps1", C.c_float),
                ("eps2", C.c_float), ("w1", C.c_int32), ("w2", C.c_int32), ("smooth_window", C.c_int32),
                ("early_stop", C.c_int32), ("dtf_format", C.c_int32), ("e_max", C.c_int32), ("z_min", C.c_float),
                ("device", C.c_int32), ("stream", C.c_void_p), ("pair_budget", C.c_int32),
                ("subsample_seed", C.c_uint64), ("stop_rule", C.c_int32), ("w_loss", C.c_int32),
                ("eps_loss", C.c_float), ("joint_phase", C.c_int32), ("weight_decay", C.c_float),
                ("mem_pool", C.c_void_p)]


class EpoError(RuntimeError):
    def __init__(self, status: int, where: str, msg: str):
        super().__init__(f"{where}: {_STATUS.get(status, status)}: {msg}")
        self.status = status


def load_library() -> C.CDLL:
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2607_00579_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, i32p, f32p = C.c_void_p, C.c_void_p, C.c_void_p
    L.epo_config_default.argtypes = [C.POINTER(EpoConfig)]
    L.epo_create.argtypes = [C.POINTER(EpoConfig), C.POINTER(vp)]
    L.epo_destroy.argtypes = [vp]; L.epo_destroy.restype = None
    L.epo_set_views.argtypes = [vp, f32p, f32p, f32p, vp]
    L.epo_extract_edges.argtypes = [vp, vp, C.c_int32, C.c_int32, vp]
    L.epo_extract_edges_rgb.argtypes = [vp, vp, C.c_int32, C.c_int32, vp]
    L.epo_set_pairs.argtypes = [vp, i32p, C.c_int64]
    L.epo_build_viewgraph.argtypes = [vp, C.c_int32, C.c_float, C.c_float, i32p, C.c_int64, C.POINTER(C.c_int64), i32p]
    L.epo_loss_grad.argtypes = [vp, C.c_float, f32p, f32p, i32p, f32p]
    L.epo_loss_grad_joint.argtypes = [vp, C.c_float, f32p, f32p, f32p]
    L.epo_get_joint_variables.argtypes = [vp, vp, vp, vp]
    L.epo_step.argtypes = [vp, C.c_int32, i32p, i32p]
    L.epo_get_poses.argtypes = [vp, f32p]
    L.epo_get_poses_f64.argtypes = [vp, vp]
    L.epo_reset.argtypes = [vp, f32p]
    L.epo_get_edge_counts.argtypes = [vp, i32p]
    L.epo_get_edge_list.argtypes = [vp, C.c_int32, vp, f32p]
    L.epo_get_dtf.argtypes = [vp, C.c_int32, f32p]
    L.epo_get_pair_order.argtypes = [vp, i32p, i32p]
    L.epo_get_trace.argtypes = [vp, C.c_int32, C.c_int32, f32p, f32p]
    L.epo_get_pair_subset.argtypes = [vp, C.c_int32, vp]
    L.epo_get_work.argtypes = [vp, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
    L.epo_time_loss_grad_kernel.argtypes = [vp, C.c_float, C.c_int32, C.c_int32, C.POINTER(C.c_float), C.POINTER(C.c_float)]
    L.epo_time_gather_ceiling.argtypes = L.epo_time_loss_grad_kernel.argtypes
    L.epo_edt_no_alloc.argtypes = [vp, C.c_int32, C.c_int32, vp, vp, C.c_char_p, C.c_int32]
    L.epo_get_state_size.argtypes = [vp, C.POINTER(C.c_int64)]
    L.epo_get_state.argtypes = [vp, vp, C.c_int64]
    L.epo_set_state.argtypes = [vp, vp, C.c_int64]
    L.epo_last_error.argtypes = [vp]; L.epo_last_error.restype = C.c_char_p
    L.epo_version.argtypes = []; L.epo_version.restype = C.c_char_p
    return L


_lib: Optional[C.CDLL] = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        _lib = load_library()
    return _lib


def _ptr(a, dtype=None):
    """Raw address of a numpy array or torch tensor (contiguity and dtype are the caller's contract)."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        assert a.flags.c_contiguous, "array must be C-contiguous"
        if dtype is not None:
            assert a.dtype == dtype, (a.dtype, dtype)
        return a.ctypes.data
    if hasattr(a, "data_ptr"):    # torch tensor
        assert a.is_contiguous(), "tensor must be contiguous"
        return a.data_ptr()
    raise TypeError(type(a))


def epo_config_default(**overrides) -> EpoConfig:
    cfg = EpoConfig()
    st = lib().epo_config_default(C.byref(cfg))
    if st != EPO_OK:
        raise EpoError(st, "epo_config_default", "")
    for k, v in overrides.items():
        setattr(cfg, k, v)
    return cfg


EDT_NO_ALLOC_MAX_PIXELS = 512 * 1024     # EPO_EDT_NO_ALLOC_MAX_PIXELS of include/epo.h


def edt_no_alloc(edges, dtf, stream: int = 0):
    """epo_edt_no_alloc: distance field of one [H][W] u8 edge map into the [H][W] fp32 tensor `dtf`, both CUDA tensors of
    the current device that the CALLER allocated -- this call takes no device memory of its own (see include/epo.h for
    who needs that, the 512 Ki-pixel limit and the rule that overlapping calls on one GPU race).  `stream` is a raw
    cudaStream_t (0 = default stream); the call does not synchronise."""
    H, W = int(edges.shape[0]), int(edges.shape[1])
    assert tuple(dtf.shape) == (H, W), (tuple(dtf.shape), (H, W))
    buf = C.create_string_buffer(256)
    st = lib().epo_edt_no_alloc(_ptr(edges, np.uint8), W, H, _ptr(dtf, np.float32), stream, buf, len(buf))
    if st != EPO_OK:
        raise EpoError(st, "epo_edt_no_alloc", buf.value.decode())


class Epo:
    """One epo_ctx.  Methods mirror the C entry points one to one."""

    def __init__(self, cfg: EpoConfig):
        self._h = C.c_void_p()
        self.cfg = cfg
        st = lib().epo_create(C.byref(cfg), C.byref(self._h))
        if st != EPO_OK:
            raise EpoError(st, "epo_create", "no context (is a CUDA device present? there is no CPU fallback)")
        self.N, self.W, self.H = cfg.n_views, cfg.width, cfg.height
        self.P = 0

    def _check(self, st: int, where: str):
        if st != EPO_OK:
            raise EpoError(st, where, lib().epo_last_error(self._h).decode())

    def destroy(self):
        if self._h:
            lib().epo_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    # ---- the six calls of the north star -----------------------------------------------------
    def set_views(self, K, poses, depth, edges):
        self._check(lib().epo_set_views(self._h, _ptr(K, np.float32), _ptr(poses, np.float32),
                                        _ptr(depth, np.float32), _ptr(edges, np.uint8)), "epo_set_views")
        self.P = 0

    def extract_edges(self, images, low: int, high: int, out=None):
        """Canny edge maps [N][H][W] u8 (1 / 0) of 8-bit grey images (numpy or torch, host or CUDA)."""
        if out is None:
            out = np.zeros((self.N, self.H, self.W), np.uint8)
        self._check(lib().epo_extract_edges(self._h, _ptr(images), int(low), int(high), _ptr(out)), "epo_extract_edges")
        return out

    def extract_edges_rgb(self, rgb, low: int, high: int, out=None):
        """Canny edge maps [N][H][W] u8 of [N][H][W][3] 8-bit colour images (BT.601 luma, then extract_edges)."""
        if out is None:
            out = np.zeros((self.N, self.H, self.W), np.uint8)
        self._check(lib().epo_extract_edges_rgb(self._h, _ptr(rgb), int(low), int(high), _ptr(out)), "epo_extract_edges_rgb")
        return out

    def build_viewgraph(self, stride: int = 8, tau: float = 3.0, min_frac: float = 0.125, want_counts: bool = False):
        """Directed pair list [P][2] (int32) of the cycle-consistent viewgraph at the current poses (+ counts [N][N][2])."""
        n = C.c_int64(0)
        cap = self.N * (self.N - 1)
        pairs = np.zeros((max(cap, 1), 2), np.int32)
        counts = np.zeros((self.N, self.N, 2), np.int32) if want_counts else None
        self._check(lib().epo_build_viewgraph(self._h, int(stride), C.c_float(tau), C.c_float(min_frac), _ptr(pairs), cap,
                                              C.byref(n), _ptr(counts)), "epo_build_viewgraph")
        pairs = np.ascontiguousarray(pairs[: n.value])
        return (pairs, counts) if want_counts else pairs

    def set_pairs(self, pairs):
        n = int(pairs.shape[0])
        self._check(lib().epo_set_pairs(self._h, _ptr(pairs, np.int32), n), "epo_set_pairs")
        self.P = n

    def loss_grad(self, lam: float, want_pairs: bool = True, want_grad: bool = True):
        """Host-side convenience: returns dict(loss, pair_loss, pair_valid, grad) as numpy arrays."""
        loss = np.zeros(1, np.float32)
        pl = np.zeros(self.P, np.float32) if want_pairs else None
        pv = np.zeros(self.P, np.int32) if want_pairs else None
        g = np.zeros((self.N, 6), np.float32) if want_grad else None
        self.loss_grad_into(lam, loss, pl, pv, g)
        return dict(loss=float(loss[0]), pair_loss=pl, pair_valid=pv, grad=g)

    def loss_grad_into(self, lam: float, loss, pair_loss=None, pair_valid=None, grad=None):
        """Raw call: outputs may be numpy arrays or torch tensors (device outputs do not synchronise)."""
        self._check(lib().epo_loss_grad(self._h, C.c_float(lam), _ptr(loss), _ptr(pair_loss), _ptr(pair_valid),
                                        _ptr(grad)), "epo_loss_grad")

    def loss_grad_joint(self, lam: float):
        """Joint-phase gradients: dict(loss, g_logf [N], g_depth [N][H][W]) as numpy arrays."""
        loss = np.zeros(1, np.float32); gf = np.zeros(self.N, np.float32)
        gz = np.zeros((self.N, self.H, self.W), np.float32)
        self._check(lib().epo_loss_grad_joint(self._h, C.c_float(lam), _ptr(loss), _ptr(gf), _ptr(gz)), "epo_loss_grad_joint")
        return dict(loss=float(loss[0]), g_logf=gf, g_depth=gz)

    def get_joint_variables(self):
        """(gamma [N], alpha [N][H][W], beta [N][H][W]) as float64 numpy arrays (cfg.joint_phase = 1)."""
        g = np.zeros(self.N); a = np.zeros((self.N, self.H, self.W)); b = np.zeros((self.N, self.H, self.W))
        self._check(lib().epo_get_joint_variables(self._h, _ptr(g), _ptr(a), _ptr(b)), "epo_get_joint_variables")
        return g, a, b

    def step(self, n_iters: int, sync: bool = True):
        """Runs up to n_iters iterations; returns (iters_done, phase) if sync else None."""
        if not sync:
            self._check(lib().epo_step(self._h, n_iters, None, None), "epo_step")
            return None
        out = np.zeros(2, np.int32)
        self._check(lib().epo_step(self._h, n_iters, out.ctypes.data, out.ctypes.data + 4), "epo_step")
        return int(out[0]), int(out[1])

    def get_poses(self, out=None):
        if out is None:
            out = np.zeros((self.N, 12), np.float32)
        self._check(lib().epo_get_poses(self._h, _ptr(out)), "epo_get_poses")
        return out

    # ---- extras --------------------------------------------------------------------------------
    def get_poses_f64(self):
        out = np.zeros((self.N, 12), np.float64)
        self._check(lib().epo_get_poses_f64(self._h, _ptr(out)), "epo_get_poses_f64")
        return out

    def reset(self, poses=None):
        self._check(lib().epo_reset(self._h, _ptr(poses, np.float32)), "epo_reset")

    def get_state(self):
        """The optimiser state as a uint8 numpy array (epo_get_state): restore with set_state into a context with the same
        configuration, views and pairs."""
        n = C.c_int64(0)
        self._check(lib().epo_get_state_size(self._h, C.byref(n)), "epo_get_state_size")
        blob = np.zeros(n.value, np.uint8)
        self._check(lib().epo_get_state(self._h, _ptr(blob), n.value), "epo_get_state")
        return blob

    def set_state(self, blob):
        self._check(lib().epo_set_state(self._h, _ptr(blob), int(blob.size if isinstance(blob, np.ndarray) else blob.numel())),
                    "epo_set_state")

    def get_edge_counts(self):
        off = np.zeros(self.N + 1, np.int32)
        self._check(lib().epo_get_edge_counts(self._h, _ptr(off)), "epo_get_edge_counts")
        return off

    def get_edge_list(self, view: int, count: int):
        uv = np.zeros((count, 2), np.uint16); z = np.zeros(count, np.float32)
        self._check(lib().epo_get_edge_list(self._h, view, _ptr(uv), _ptr(z)), "epo_get_edge_list")
        return uv, z

    def get_dtf(self, view: int):
        out = np.zeros((self.H, self.W), np.float32)
        self._check(lib().epo_get_dtf(self._h, view, _ptr(out)), "epo_get_dtf")
        return out

    def get_pair_order(self):
        cp = np.zeros((self.P, 2), np.int32); perm = np.zeros(self.P, np.int32)
        self._check(lib().epo_get_pair_order(self._h, _ptr(cp), _ptr(perm)), "epo_get_pair_order")
        return cp, perm

    def get_trace(self, first: int, count: int):
        loss = np.zeros(count, np.float32); th = np.zeros(count, np.float32)
        self._check(lib().epo_get_trace(self._h, first, count, _ptr(loss), _ptr(th)), "epo_get_trace")
        return loss, th

    def time_loss_grad_kernel(self, lam: float, reps: int, flush_l2: bool):
        """(mean ms, min ms) of the fused kernel alone, CUDA events on the library's stream."""
        a = C.c_float(); b = C.c_float()
        self._check(lib().epo_time_loss_grad_kernel(self._h, C.c_float(lam), reps, int(flush_l2), C.byref(a), C.byref(b)),
                    "epo_time_loss_grad_kernel")
        return float(a.value), float(b.value)

    def time_gather_ceiling(self, lam: float, reps: int, flush_l2: bool):
        """(mean ms, min ms) of the fused kernel's memory side alone (its gather roofline on this workload)."""
        a = C.c_float(); b = C.c_float()
        self._check(lib().epo_time_gather_ceiling(self._h, C.c_float(lam), reps, int(flush_l2), C.byref(a), C.byref(b)),
                    "epo_time_gather_ceiling")
        return float(a.value), float(b.value)

    def get_pair_subset(self, step: int):
        """Boolean mask (caller's pair order) of the pairs iteration `step` evaluates."""
        flags = np.zeros(self.P, np.uint8)
        self._check(lib().epo_get_pair_subset(self._h, int(step), _ptr(flags)), "epo_get_pair_subset")
        return flags.astype(bool)

    def get_work(self):
        r = C.c_int64(); k = C.c_int64()
        self._check(lib().epo_get_work(self._h, C.byref(r), C.byref(k)), "epo_get_work")
        return int(r.value), int(k.value)
