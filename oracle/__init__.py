"""ctypes front-end of the CPU oracle (oracle/epo_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, by __graft_entry__.smoke() and by bench.py's
cpu_baseline / --impl reference legs.  The product package (paper_2607_00579_b200) never imports
this module and this module never imports the product package.  This file only marshals numpy arrays
into the C functions; all arithmetic of the method lives in epo_oracle.c, each function citing the
passage of PAPER.md it follows.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "epo_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile epo_oracle.c with gcc (-O2, no fast-math, no FMA contraction, OpenMP over pairs).
    EPO_ORACLE_SANITIZE=1 builds and loads an AddressSanitizer + UndefinedBehaviorSanitizer instance instead
    (liboracle_san.so; run python with LD_PRELOAD=$(gcc -print-file-name=libasan.so): profiles/r2_sanitizer.md)."""
    san = os.environ.get("EPO_ORACLE_SANITIZE", "") not in ("", "0")
    lib = os.path.join(_HERE, "liboracle_san.so") if san else _LIB
    if force or not os.path.exists(lib) or os.path.getmtime(lib) < os.path.getmtime(_SRC):
        tmp = lib + ".%d.tmp" % os.getpid()
        flags = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-omit-frame-pointer"] if san else ["-O2"]
        subprocess.check_call(["gcc"] + flags + ["-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, lib)
    return lib


class _Cfg(C.Structure):
    _fields_ = [("huber_delta", C.c_double), ("clamp_start", C.c_double), ("clamp_end", C.c_double),
                ("clamp_steps", C.c_int32), ("lr_max", C.c_double), ("warmup_steps", C.c_int32),
                ("max_steps", C.c_int32), ("beta1", C.c_double), ("beta2", C.c_double),
                ("adam_eps", C.c_double), ("eps1", C.c_double), ("eps2", C.c_double), ("w1", C.c_int32),
                ("w2", C.c_int32), ("smooth_window", C.c_int32), ("early_stop", C.c_int32),
                ("z_min", C.c_double), ("coord_fp32", C.c_int32), ("stop_rule", C.c_int32), ("w_loss", C.c_int32),
                ("eps_loss", C.c_double)]


@dataclass
class Config:
    """Hyper-parameters with the paper's values and the readings S1, S10."""
    huber_delta: float = 1.0
    clamp_start: float = 10.0
    clamp_end: float = 6.0
    clamp_steps: int = 1000
    lr_max: float = 3e-3
    warmup_steps: int = 25
    max_steps: int = 2000
    beta1: float = 0.9
    beta2: float = 0.999
    adam_eps: float = 1e-8
    eps1: float = 0.5
    eps2: float = 0.1
    w1: int = 25
    w2: int = 50
    smooth_window: int = 1
    early_stop: int = 0
    z_min: float = 1e-6
    coord_fp32: int = 0      # 1: projected positions decided in fp32 (reading P1)
    stop_rule: int = 0       # second-stage rule: 0 pose-based (the paper's), 1 loss-based
    w_loss: int = 100
    eps_loss: float = 5e-4

    def c(self) -> _Cfg:
        return _Cfg(**{f[0]: getattr(self, f[0]) for f in _Cfg._fields_})


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t)) if a is not None else None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_lambda.restype = C.c_double
        L.orc_lambda.argtypes = [C.c_int, C.c_double, C.c_double, C.c_int]
        L.orc_lr.restype = C.c_double
        L.orc_lr.argtypes = [C.c_int, C.c_double, C.c_int, C.c_int]
        L.orc_delta_R_deg.restype = C.c_double
        L.orc_delta_t_deg.restype = C.c_double
        L.orc_percentile.restype = C.c_double
        L.orc_percentile.argtypes = [C.c_int, C.POINTER(C.c_double), C.c_double]
        L.orc_theta95.restype = C.c_double
        L.orc_round_to_half.restype = C.c_float
        L.orc_round_to_half.argtypes = [C.c_float]
        L.orc_adamw.argtypes = [C.c_int64, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_double),
                                C.POINTER(C.c_double), C.c_int, C.c_double, C.c_double, C.c_double, C.c_double, C.c_double,
                                C.c_double]
        L.orc_converged_loss.argtypes = [C.POINTER(C.c_double), C.c_int, C.c_int, C.c_double]
        L.orc_converged.argtypes = [C.POINTER(C.c_double), C.c_int, C.c_int, C.c_double, C.c_int]
        L.orc_adam.argtypes = [C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_double),
                               C.c_int, C.c_double, C.c_double, C.c_double, C.c_double, C.POINTER(C.c_double)]
        L.orc_edge_list.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_uint8), C.POINTER(C.c_float), C.c_double,
                                    C.c_int, C.POINTER(C.c_uint16), C.POINTER(C.c_float)]
        L.orc_pair_loss_grad.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(C.c_uint16), C.POINTER(C.c_float),
                                         C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_double),
                                         C.POINTER(C.c_double), C.POINTER(C.c_float), C.c_double, C.c_double,
                                         C.c_double, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_int32),
                                         C.POINTER(C.c_double), C.POINTER(C.c_int32)]
        L.orc_loss_grad.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(C.c_float), C.POINTER(C.c_double),
                                    C.POINTER(C.c_int32), C.POINTER(C.c_uint16), C.POINTER(C.c_float),
                                    C.POINTER(C.c_float), C.c_int64, C.POINTER(C.c_int32), C.c_double,
                                    C.c_double, C.c_double, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_int32),
                                    C.POINTER(C.c_double), C.POINTER(C.c_int32), C.POINTER(C.c_double),
                                    C.POINTER(C.c_double)]
        L.orc_pair_event_slack.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(C.c_uint16), C.POINTER(C.c_float),
                                           C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_double),
                                           C.POINTER(C.c_double), C.POINTER(C.c_float), C.c_double, C.c_double,
                                           C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.orc_event_slack.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(C.c_float), C.POINTER(C.c_double),
                                      C.POINTER(C.c_int32), C.POINTER(C.c_uint16), C.POINTER(C.c_float),
                                      C.POINTER(C.c_float), C.c_int64, C.POINTER(C.c_int32), C.c_double, C.c_double,
                                      C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_int32), C.POINTER(C.c_double),
                                      C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_int32), C.POINTER(C.c_double)]
        L.orc_joint_slack.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(C.c_float), C.POINTER(C.c_double),
                                      C.POINTER(C.c_int32), C.POINTER(C.c_uint16), C.POINTER(C.c_float),
                                      C.POINTER(C.c_float), C.c_int64, C.POINTER(C.c_int32), C.c_double, C.c_double,
                                      C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.orc_joint_grad.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(C.c_float), C.POINTER(C.c_double),
                                     C.POINTER(C.c_int32), C.POINTER(C.c_uint16), C.POINTER(C.c_float),
                                     C.POINTER(C.c_float), C.c_int64, C.POINTER(C.c_int32), C.c_double, C.c_double,
                                     C.c_double, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.orc_run.restype = C.c_int
        L.orc_run.argtypes = [C.POINTER(_Cfg), C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_float),
                              C.POINTER(C.c_double), C.POINTER(C.c_int32), C.POINTER(C.c_uint16),
                              C.POINTER(C.c_float), C.POINTER(C.c_float), C.c_int64, C.POINTER(C.c_int32),
                              C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_double),
                              C.POINTER(C.c_double), C.POINTER(C.c_int32), C.POINTER(C.c_int32),
                              C.POINTER(C.c_double)]
        L.orc_canny_blur.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_uint8), C.POINTER(C.c_uint8)]
        L.orc_canny_sobel.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_uint8), C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
        L.orc_canny_suppress.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_int32), C.POINTER(C.c_int32), C.c_int, C.c_int,
                                         C.POINTER(C.c_uint8)]
        L.orc_canny_hysteresis.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_uint8), C.POINTER(C.c_uint8)]
        L.orc_canny.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(C.c_uint8), C.c_int, C.c_int, C.POINTER(C.c_uint8)]
        L.orc_viewgraph_counts.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(C.c_float), C.POINTER(C.c_double),
                                           C.POINTER(C.c_float), C.c_int, C.c_double, C.c_double, C.c_int,
                                           C.POINTER(C.c_int32)]
        L.orc_viewgraph_counts_slack.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(C.c_float), C.POINTER(C.c_double),
                                                 C.POINTER(C.c_float), C.c_int, C.c_double, C.c_double, C.POINTER(C.c_int32)]
        L.orc_viewgraph_pairs.restype = C.c_int64
        L.orc_viewgraph_pairs.argtypes = [C.c_int, C.POINTER(C.c_int32), C.c_double, C.POINTER(C.c_int32)]
        L.orc_subset_key.restype = C.c_uint64
        L.orc_subset_key.argtypes = [C.c_uint64, C.c_int, C.c_int64]
        L.orc_pair_subset.restype = C.c_int64
        L.orc_pair_subset.argtypes = [C.c_uint64, C.c_int, C.c_int64, C.c_int64, C.c_void_p]
        L.orc_canonical_pairs.argtypes = [C.c_int64, C.POINTER(C.c_int32), C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def set_num_threads(n: int) -> None:
    lib().orc_set_num_threads(int(n))


# ---------------------------------------------------------------------------------------------- O1
def edge_list(edges: np.ndarray, depth: np.ndarray, z_min: float = 1e-6, e_max: int = 0):
    """(uv uint16 [E,2], z float32 [E]) of one view, raster order."""
    H, W = edges.shape
    edges = np.ascontiguousarray(edges, np.uint8); depth = np.ascontiguousarray(depth, np.float32)
    uv = np.empty((H * W, 2), np.uint16); z = np.empty(H * W, np.float32)
    n = lib().orc_edge_list(W, H, _p(edges, C.c_uint8), _p(depth, C.c_float), z_min, e_max,
                            _p(uv, C.c_uint16), _p(z, C.c_float))
    return uv[:n].copy(), z[:n].copy()


def edge_lists(edges: np.ndarray, depth: np.ndarray, z_min: float = 1e-6, e_max: int = 0):
    """All views: (offsets int32 [N+1], uv [E,2], z [E])."""
    lists = [edge_list(edges[i], depth[i], z_min, e_max) for i in range(edges.shape[0])]
    off = np.zeros(len(lists) + 1, np.int32)
    off[1:] = np.cumsum([len(l[1]) for l in lists])
    uv = np.concatenate([l[0] for l in lists]) if lists else np.empty((0, 2), np.uint16)
    z = np.concatenate([l[1] for l in lists]) if lists else np.empty(0, np.float32)
    return off, np.ascontiguousarray(uv), np.ascontiguousarray(z)


# ---------------------------------------------------------------------------------------------- O2
def edt_brute(edges: np.ndarray) -> np.ndarray:
    H, W = edges.shape
    edges = np.ascontiguousarray(edges, np.uint8); out = np.empty((H, W), np.float32)
    lib().orc_edt_brute(W, H, _p(edges, C.c_uint8), _p(out, C.c_float))
    return out


def edt(edges: np.ndarray) -> np.ndarray:
    """Exact EDT of one view [H,W] or a batch [N,H,W] (separable form, exhaustive integer minima)."""
    edges = np.ascontiguousarray(edges, np.uint8)
    out = np.empty(edges.shape, np.float32)
    if edges.ndim == 2:
        H, W = edges.shape
        lib().orc_edt_separable(W, H, _p(edges, C.c_uint8), _p(out, C.c_float))
    else:
        N, H, W = edges.shape
        lib().orc_edt_batch(N, W, H, _p(edges, C.c_uint8), _p(out, C.c_float))
    return out


def round_to_half(field: np.ndarray) -> np.ndarray:
    field = np.ascontiguousarray(field, np.float32); out = np.empty_like(field)
    lib().orc_round_field_to_half(C.c_int64(field.size), _p(field, C.c_float), _p(out, C.c_float))
    return out


# ---------------------------------------------------------------------------------------------- O3
def canonical_pairs(pairs: np.ndarray):
    pairs = np.ascontiguousarray(pairs, np.int32); P = pairs.shape[0]
    out = np.empty_like(pairs); perm = np.empty(P, np.int32)
    lib().orc_canonical_pairs(P, _p(pairs, C.c_int32), _p(out, C.c_int32), _p(perm, C.c_int32))
    return out, perm


# ------------------------------------------------------------------------------------------ geometry
def _d(a, n=None):
    a = np.ascontiguousarray(a, np.float64)
    assert n is None or a.size == n
    return a


def backproject_cam(K, u, v, Z):
    K = _d(K, 4); out = np.empty(3)
    f = lib().orc_backproject_cam; f.argtypes = [C.POINTER(C.c_double), C.c_double, C.c_double, C.c_double, C.POINTER(C.c_double)]
    f(_p(K, C.c_double), u, v, Z, _p(out, C.c_double)); return out


def cam_to_world(T, x):
    T = _d(T, 12); x = _d(x, 3); out = np.empty(3)
    lib().orc_cam_to_world(_p(T, C.c_double), _p(x, C.c_double), _p(out, C.c_double)); return out


def world_to_cam(T, X):
    T = _d(T, 12); X = _d(X, 3); out = np.empty(3)
    lib().orc_world_to_cam(_p(T, C.c_double), _p(X, C.c_double), _p(out, C.c_double)); return out


def project_px(K, x):
    K = _d(K, 4); x = _d(x, 3); out = np.empty(2)
    lib().orc_project_px(_p(K, C.c_double), _p(x, C.c_double), _p(out, C.c_double)); return out


def relative_pose(Ts, Tt):
    Ts = _d(Ts, 12); Tt = _d(Tt, 12); out = np.empty(12)
    lib().orc_relative_pose(_p(Ts, C.c_double), _p(Tt, C.c_double), _p(out, C.c_double)); return out


# ------------------------------------------------------------------------------------------- O4-O6
def pair_loss_grad(uv, z, Ks, Kt, Ts, Tt, dtf_t, lam, delta=1.0, z_min=1e-6, coord_fp32=0):
    """One directed pair: (sum_rho, n_valid, G[12] = [tgt(v,w), src(v,w)] un-normalised, near[2])."""
    H, W = dtf_t.shape
    uv = np.ascontiguousarray(uv, np.uint16); z = np.ascontiguousarray(z, np.float32)
    dtf_t = np.ascontiguousarray(dtf_t, np.float32)
    S = C.c_double(); nv = C.c_int32(); G = np.empty(12); near = np.zeros(2, np.int32)
    lib().orc_pair_loss_grad(W, H, len(z), _p(uv, C.c_uint16), _p(z, C.c_float), _p(_d(Ks, 4), C.c_double),
                             _p(_d(Kt, 4), C.c_double), _p(_d(Ts, 12), C.c_double), _p(_d(Tt, 12), C.c_double),
                             _p(dtf_t, C.c_float), lam, delta, z_min, coord_fp32, C.byref(S), C.byref(nv),
                             _p(G, C.c_double), _p(near, C.c_int32))
    return S.value, nv.value, G, near


@dataclass
class Problem:
    """Preprocessed inputs of the loss: edge lists and distance fields of all views."""
    W: int
    H: int
    K: np.ndarray          # [N,4] float32
    edge_off: np.ndarray   # [N+1] int32
    uv: np.ndarray         # [E,2] uint16
    z: np.ndarray          # [E] float32
    dtf: np.ndarray        # [N,H,W] float32

    @property
    def n_views(self):
        return self.K.shape[0]


def preprocess(K, depth, edges, z_min=1e-6, e_max=0, half=False) -> Problem:
    N, H, W = edges.shape
    off, uv, z = edge_lists(edges, depth, z_min, e_max)
    dtf = edt(edges)
    if half:
        dtf = round_to_half(dtf)
    return Problem(W, H, np.ascontiguousarray(K, np.float32), off, uv, z, dtf)


def loss_grad(prob: Problem, poses, pairs, lam, delta=1.0, z_min=1e-6, want_pair_G=False, coord_fp32=0):
    """Returns dict(loss, pair_loss [P], pair_valid [P], grad [N,6], near [P,2], pair_G [P,12]?)."""
    N = prob.n_views
    poses = np.ascontiguousarray(np.asarray(poses, np.float64).reshape(N, 12))
    pairs = np.ascontiguousarray(pairs, np.int32); P = pairs.shape[0]
    pl = np.empty(P); pv = np.empty(P, np.int32); near = np.zeros((P, 2), np.int32)
    pG = np.empty((P, 12)) if want_pair_G else None
    grad = np.empty((N, 6)); L = C.c_double()
    lib().orc_loss_grad(N, prob.W, prob.H, _p(prob.K, C.c_float), _p(poses, C.c_double),
                        _p(prob.edge_off, C.c_int32), _p(prob.uv, C.c_uint16), _p(prob.z, C.c_float),
                        _p(prob.dtf, C.c_float), P, _p(pairs, C.c_int32), lam, delta, z_min, coord_fp32,
                        _p(pl, C.c_double), _p(pv, C.c_int32), _p(pG, C.c_double), _p(near, C.c_int32),
                        _p(grad, C.c_double), C.byref(L))
    return dict(loss=L.value, pair_loss=pl, pair_valid=pv, grad=grad, near=near, pair_G=pG)


def pair_event_slack(uv, z, Ks, Kt, Ts, Tt, dtf_t, lam, delta=1.0, z_min=1e-6):
    """One directed pair: what a correct binary32 evaluation may decide differently (see orc_pair_event_slack).
    Returns dict(E_t, E_s, E_rho, k_out, k_in, flagged, check [14] = S, n, G[12] through the slack routine)."""
    H, W = dtf_t.shape
    uv = np.ascontiguousarray(uv, np.uint16); z = np.ascontiguousarray(z, np.float32)
    dtf_t = np.ascontiguousarray(dtf_t, np.float32)
    out = np.zeros(8); chk = np.zeros(14)
    lib().orc_pair_event_slack(W, H, len(z), _p(uv, C.c_uint16), _p(z, C.c_float), _p(_d(Ks, 4), C.c_double),
                               _p(_d(Kt, 4), C.c_double), _p(_d(Ts, 12), C.c_double), _p(_d(Tt, 12), C.c_double),
                               _p(dtf_t, C.c_float), lam, delta, z_min, _p(out, C.c_double), _p(chk, C.c_double))
    return dict(E_t=out[0], E_s=out[1], E_rho=out[2], k_out=int(out[3]), k_in=int(out[4]), flagged=int(out[5]), Q_t=out[6],
                Q_s=out[7], check=chk)


def event_slack(prob: Problem, poses, pairs, lam, ref=None, delta=1.0, z_min=1e-6):
    """Bounds on what a correct binary32 evaluation may differ by from `ref` = loss_grad(..., want_pair_G=True) (all
    double) through its discrete decisions: dict(cam [N] on the 2-norm of each camera's gradient, pair_loss [P],
    k_out [P], k_in [P] on the valid counts, flagged [P], rss [N] = root-sum-square of the terms of each camera's
    gradient: its scale before cancellation, reading T2)."""
    N = prob.n_views
    poses = np.ascontiguousarray(np.asarray(poses, np.float64).reshape(N, 12))
    pairs = np.ascontiguousarray(pairs, np.int32); P = pairs.shape[0]
    if ref is None or ref.get("pair_G") is None:
        ref = loss_grad(prob, poses, pairs, lam, delta, z_min, want_pair_G=True)
    cam = np.zeros(N); pls = np.zeros(P); fl = np.zeros((P, 3), np.int32); rss = np.zeros(N)
    pl = np.ascontiguousarray(ref["pair_loss"], np.float64); pv = np.ascontiguousarray(ref["pair_valid"], np.int32)
    pG = np.ascontiguousarray(ref["pair_G"], np.float64)
    lib().orc_event_slack(N, prob.W, prob.H, _p(prob.K, C.c_float), _p(poses, C.c_double), _p(prob.edge_off, C.c_int32),
                          _p(prob.uv, C.c_uint16), _p(prob.z, C.c_float), _p(prob.dtf, C.c_float), P, _p(pairs, C.c_int32),
                          C.c_double(lam), C.c_double(delta), C.c_double(z_min), _p(pl, C.c_double), _p(pv, C.c_int32),
                          _p(pG, C.c_double), _p(cam, C.c_double), _p(pls, C.c_double), _p(fl, C.c_int32), _p(rss, C.c_double))
    return dict(cam=cam, pair_loss=pls, k_out=fl[:, 0].copy(), k_in=fl[:, 1].copy(), flagged=fl[:, 2].copy(), rss=rss)


def joint_grad(prob: Problem, poses, pairs, lam, delta=1.0, z_min=1e-6, coord_fp32=0):
    """Joint-phase gradients (Eq. 4-5): (d L / d ln f_c [N], d L / d Z_e [E] in edge-list order)."""
    N = prob.n_views
    poses = np.ascontiguousarray(np.asarray(poses, np.float64).reshape(N, 12))
    pairs = np.ascontiguousarray(pairs, np.int32); P = pairs.shape[0]
    g_f = np.zeros(N); g_z = np.zeros(int(prob.edge_off[-1]))
    lib().orc_joint_grad(N, prob.W, prob.H, _p(prob.K, C.c_float), _p(poses, C.c_double), _p(prob.edge_off, C.c_int32),
                         _p(prob.uv, C.c_uint16), _p(prob.z, C.c_float), _p(prob.dtf, C.c_float), P, _p(pairs, C.c_int32),
                         C.c_double(lam), C.c_double(delta), C.c_double(z_min), int(coord_fp32), _p(g_f, C.c_double),
                         _p(g_z, C.c_double))
    return g_f, g_z


def joint_slack(prob: Problem, poses, pairs, lam, delta=1.0, z_min=1e-6):
    """Event slack of the joint-phase gradients (see orc_joint_slack): dict(logf [N], logf_rss [N], gz [E])."""
    N = prob.n_views
    poses = np.ascontiguousarray(np.asarray(poses, np.float64).reshape(N, 12))
    pairs = np.ascontiguousarray(pairs, np.int32); P = pairs.shape[0]
    sf = np.zeros(N); rf = np.zeros(N); sz = np.zeros(int(prob.edge_off[-1]))
    lib().orc_joint_slack(N, prob.W, prob.H, _p(prob.K, C.c_float), _p(poses, C.c_double), _p(prob.edge_off, C.c_int32),
                          _p(prob.uv, C.c_uint16), _p(prob.z, C.c_float), _p(prob.dtf, C.c_float), P, _p(pairs, C.c_int32),
                          C.c_double(lam), C.c_double(delta), C.c_double(z_min), _p(sf, C.c_double), _p(rf, C.c_double),
                          _p(sz, C.c_double))
    return dict(logf=sf, logf_rss=rf, gz=sz)


# ---------------------------------------------------------------------------------------------- O7
def _u8p(a):
    return a.ctypes.data_as(C.POINTER(C.c_uint8))


def rgb_to_grey(rgb: np.ndarray) -> np.ndarray:
    """[..., 3] uint8 -> [...] uint8, reading C7 (BT.601 luma in 8-bit fixed point)."""
    rgb = np.ascontiguousarray(rgb, np.uint8); assert rgb.shape[-1] == 3
    out = np.zeros(rgb.shape[:-1], np.uint8)
    lib().orc_rgb_to_grey.argtypes = [C.c_int64, C.POINTER(C.c_uint8), C.POINTER(C.c_uint8)]
    lib().orc_rgb_to_grey(C.c_int64(out.size), _u8p(rgb), _u8p(out)); return out


def canny_blur(img: np.ndarray) -> np.ndarray:
    img = np.ascontiguousarray(img, np.uint8); H, W = img.shape
    out = np.zeros_like(img); lib().orc_canny_blur(W, H, _u8p(img), _u8p(out)); return out


def canny_sobel(b: np.ndarray):
    b = np.ascontiguousarray(b, np.uint8); H, W = b.shape
    gx = np.zeros((H, W), np.int32); gy = np.zeros((H, W), np.int32)
    lib().orc_canny_sobel(W, H, _u8p(b), _p(gx, C.c_int32), _p(gy, C.c_int32)); return gx, gy


def canny_suppress(gx, gy, low: int, high: int) -> np.ndarray:
    gx = np.ascontiguousarray(gx, np.int32); gy = np.ascontiguousarray(gy, np.int32); H, W = gx.shape
    c = np.zeros((H, W), np.uint8)
    lib().orc_canny_suppress(W, H, _p(gx, C.c_int32), _p(gy, C.c_int32), int(low), int(high), _u8p(c)); return c


def canny_hysteresis(cand: np.ndarray) -> np.ndarray:
    cand = np.ascontiguousarray(cand, np.uint8); H, W = cand.shape
    e = np.zeros((H, W), np.uint8); lib().orc_canny_hysteresis(W, H, _u8p(cand), _u8p(e)); return e


def canny(images: np.ndarray, low: int, high: int) -> np.ndarray:
    """Edge maps [N][H][W] (1 / 0) of 8-bit images: the Canny detector [4], readings C1-C6."""
    images = np.ascontiguousarray(images, np.uint8)
    if images.ndim == 2:
        return canny(images[None], low, high)[0]
    N, H, W = images.shape
    e = np.zeros((N, H, W), np.uint8)
    lib().orc_canny(N, W, H, _u8p(images), int(low), int(high), _u8p(e)); return e


def viewgraph_counts(K, poses, depth, stride=8, tau=3.0, z_min=1e-6, coord_fp32=0) -> np.ndarray:
    """[N][N][2] = (consistent, usable) grid points of the cycle i -> j -> i."""
    K = np.ascontiguousarray(K, np.float32); poses = np.ascontiguousarray(poses, np.float64).reshape(-1, 12)
    depth = np.ascontiguousarray(depth, np.float32)
    N, H, W = depth.shape
    counts = np.zeros((N, N, 2), np.int32)
    lib().orc_viewgraph_counts(N, W, H, _p(K, C.c_float), _p(poses, C.c_double), _p(depth, C.c_float), int(stride),
                               C.c_double(tau), C.c_double(z_min), int(coord_fp32), _p(counts, C.c_int32))
    return counts


def viewgraph_counts_slack(K, poses, depth, stride=8, tau=3.0, z_min=1e-6) -> np.ndarray:
    """[N][N][3] = (consistent, usable, uncertain) of the cycle i -> j -> i, all double: `uncertain` counts the grid points a
    correct binary32 evaluation may decide differently (reading T1)."""
    K = np.ascontiguousarray(K, np.float32); poses = np.ascontiguousarray(poses, np.float64).reshape(-1, 12)
    depth = np.ascontiguousarray(depth, np.float32)
    N, H, W = depth.shape
    counts = np.zeros((N, N, 3), np.int32)
    lib().orc_viewgraph_counts_slack(N, W, H, _p(K, C.c_float), _p(poses, C.c_double), _p(depth, C.c_float), int(stride),
                                     C.c_double(tau), C.c_double(z_min), _p(counts, C.c_int32))
    return counts


def viewgraph_pairs_robust(counts3: np.ndarray, min_frac=0.125):
    """(certain, possible): boolean [N][N] masks of the unordered pairs i < j that are valid whatever the uncertain grid
    points decide, and of those that are valid for at least one decision of them (rule V7 on count +- uncertain)."""
    c = counts3.astype(np.int64); N = c.shape[0]
    lo = (c[..., 0] - c[..., 2]).astype(np.float64) >= np.float64(min_frac) * c[..., 1]
    hi = (c[..., 0] + c[..., 2]).astype(np.float64) >= np.float64(min_frac) * c[..., 1]
    iu = np.triu(np.ones((N, N), bool), 1)
    return (lo & lo.T) & iu, (hi & hi.T) & iu


def viewgraph_pairs(counts: np.ndarray, min_frac=0.125) -> np.ndarray:
    """Directed pair list [(i, j), (j, i) for valid i < j] from the cycle counts."""
    counts = np.ascontiguousarray(counts, np.int32); N = counts.shape[0]
    n = lib().orc_viewgraph_pairs(N, _p(counts, C.c_int32), C.c_double(min_frac), None)
    pairs = np.zeros((max(n, 1), 2), np.int32)
    lib().orc_viewgraph_pairs(N, _p(counts, C.c_int32), C.c_double(min_frac), _p(pairs, C.c_int32))
    return pairs[:n]


def subset_key(seed: int, step: int, p: int) -> int:
    """key(step, p) of the stochastic pair sub-sampling: a SplitMix64 output, see epo_oracle.c."""
    return int(lib().orc_subset_key(C.c_uint64(seed & 0xFFFFFFFFFFFFFFFF), int(step), C.c_int64(p)))


def pair_subset(seed: int, step: int, n_pairs: int, budget: int) -> np.ndarray:
    """Boolean mask (caller's pair order) of the fresh uniform random subset S of step `step`, |S| = min(P, M)
    (PAPER.md:465-474, 500)."""
    flags = np.zeros(n_pairs, np.uint8)
    n = lib().orc_pair_subset(C.c_uint64(seed & 0xFFFFFFFFFFFFFFFF), int(step), C.c_int64(n_pairs), C.c_int64(budget),
                              flags.ctypes.data_as(C.c_void_p))
    assert n == (n_pairs if budget <= 0 or n_pairs <= budget else budget)
    return flags.astype(bool)


def lam_schedule(s, cfg: Config = Config()):
    return lib().orc_lambda(s, cfg.clamp_start, cfg.clamp_end, cfg.clamp_steps)


def lr_schedule(s, cfg: Config = Config()):
    return lib().orc_lr(s, cfg.lr_max, cfg.warmup_steps, cfg.max_steps)


def se3_exp(eps):
    eps = _d(eps, 6); out = np.empty(12)
    lib().orc_se3_exp(_p(eps, C.c_double), _p(out, C.c_double)); return out


def se3_compose(E, T):
    E = _d(E, 12); T = _d(T, 12); out = np.empty(12)
    lib().orc_se3_compose(_p(E, C.c_double), _p(T, C.c_double), _p(out, C.c_double)); return out


def adam(g, m, v, s, lr, beta1=0.9, beta2=0.999, adam_eps=1e-8):
    """In-place moment update; returns the increment."""
    g = _d(g); out = np.empty_like(g)
    assert m.dtype == np.float64 and v.dtype == np.float64 and m.flags.c_contiguous and v.flags.c_contiguous
    lib().orc_adam(g.size, _p(g, C.c_double), _p(m, C.c_double), _p(v, C.c_double), s, lr, beta1, beta2,
                   adam_eps, _p(out, C.c_double))
    return out


def adamw(p, g, m, v, t, lr, beta1=0.9, beta2=0.999, adam_eps=1e-8, wd=0.01, p_id=0.0):
    """In-place AdamW step number t (1-based) of one variable group, decay towards p_id (reading J6)."""
    g = _d(g)
    for a in (p, m, v):
        assert a.dtype == np.float64 and a.flags.c_contiguous and a.size == g.size
    lib().orc_adamw(C.c_int64(g.size), _p(p, C.c_double), _p(g, C.c_double), _p(m, C.c_double), _p(v, C.c_double), int(t),
                    C.c_double(lr), C.c_double(beta1), C.c_double(beta2), C.c_double(adam_eps), C.c_double(wd), C.c_double(p_id))


# ---------------------------------------------------------------------------------------------- O8
def delta_R_deg(Tcur, Tprev):
    lib().orc_delta_R_deg.argtypes = [C.POINTER(C.c_double)] * 2
    return lib().orc_delta_R_deg(_p(_d(Tcur, 12), C.c_double), _p(_d(Tprev, 12), C.c_double))


def delta_t_deg(Tcur, Tprev):
    lib().orc_delta_t_deg.argtypes = [C.POINTER(C.c_double)] * 2
    return lib().orc_delta_t_deg(_p(_d(Tcur, 12), C.c_double), _p(_d(Tprev, 12), C.c_double))


def percentile(x, q):
    x = _d(x); return lib().orc_percentile(x.size, _p(x, C.c_double), q)


def theta95(cur, prev):
    cur = _d(cur); prev = _d(prev)
    lib().orc_theta95.argtypes = [C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    return lib().orc_theta95(cur.size // 12, _p(cur, C.c_double), _p(prev, C.c_double))


def converged_loss(loss, s, w, eps) -> bool:
    """The loss-based stopping rule at step s: relative loss change below eps for w consecutive steps."""
    loss = np.ascontiguousarray(loss, np.float64)
    return bool(lib().orc_converged_loss(_p(loss, C.c_double), int(s), int(w), C.c_double(eps)))


def converged(theta, s, w, eps, smooth=1) -> bool:
    theta = _d(theta)
    return bool(lib().orc_converged(_p(theta, C.c_double), s, w, eps, smooth))


class Optimizer:
    """State of the loop of Alg. 2 (poses, Adam moments, step, phase, theta history, loss trace)."""

    def __init__(self, prob: Problem, poses_init, pairs, cfg: Config = Config()):
        self.prob, self.cfg = prob, cfg
        N = prob.n_views
        self.poses = np.ascontiguousarray(np.asarray(poses_init, np.float32).astype(np.float64).reshape(N, 12))
        self.pairs = np.ascontiguousarray(pairs, np.int32)
        self.m = np.zeros((N, 6)); self.v = np.zeros((N, 6))
        self.theta = np.zeros(cfg.max_steps); self.loss = np.zeros(cfg.max_steps)
        self.step = C.c_int32(0); self.phase = C.c_int32(0)

    def run(self, n_iters: int, log_poses: bool = False):
        N = self.prob.n_views
        log = np.empty((n_iters, N, 12)) if log_poses else None
        c = self.cfg.c()
        done = lib().orc_run(C.byref(c), n_iters, N, self.prob.W, self.prob.H, _p(self.prob.K, C.c_float),
                             _p(self.poses, C.c_double), _p(self.prob.edge_off, C.c_int32),
                             _p(self.prob.uv, C.c_uint16), _p(self.prob.z, C.c_float), _p(self.prob.dtf, C.c_float),
                             self.pairs.shape[0], _p(self.pairs, C.c_int32), _p(self.m, C.c_double),
                             _p(self.v, C.c_double), _p(self.theta, C.c_double), _p(self.loss, C.c_double),
                             C.byref(self.step), C.byref(self.phase), _p(log, C.c_double))
        return done, (log[:done] if log_poses else None)
