"""Seeded synthetic scenes shaped like the paper's workloads (BASELINE.json configs).

The arrays produced here (K, poses, depth maps, edge masks, pair lists) are the INPUTS handed to both
the CPU oracle and the CUDA library.  This module renders them with closed-form ray / plane / box and
point / segment arithmetic; it contains none of the EPO method (no distance transform, no loss, no
gradient, no optimiser) and imports neither `oracle/` nor the CUDA package.

Conventions: OpenCV camera axes (x right, y down, z forward); poses are world-to-camera [R|t],
x_cam = R X_w + t; K = (fx, fy, cx, cy); depth is z-depth at integer pixel
positions; pixel (u, v) is the sample position (u, v) itself (no half-pixel offset).
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional

import numpy as np

from .rng import SplitMix64

BASE_SEED = 260700579 * 10


@dataclasses.dataclass
class Scene:
    name: str
    W: int
    H: int
    K: np.ndarray            # [N,4] float32 (fx, fy, cx, cy)
    poses_gt: np.ndarray     # [N,12] float64, row-major 3x4 [R|t]
    poses_init: np.ndarray   # [N,12] float32
    depth: np.ndarray        # [N,H,W] float32 (predicted depth = GT with the config's noise)
    edges: np.ndarray        # [N,H,W] uint8, nonzero = edge
    pairs: np.ndarray        # [P,2] int32 (source, target)
    meta: dict

    @property
    def n_views(self) -> int:
        return self.K.shape[0]


# ------------------------------------------------------------------------------------------------
# cameras
# ------------------------------------------------------------------------------------------------
def look_at(c: np.ndarray, target: np.ndarray, up=(0.0, 0.0, 1.0)) -> np.ndarray:
    """World-to-camera 3x4 [R|t] of a camera at `c` looking at `target` (z-up world, OpenCV axes)."""
    f = np.asarray(target, float) - np.asarray(c, float)
    f = f / np.linalg.norm(f)
    r = np.cross(f, np.asarray(up, float))
    r = r / np.linalg.norm(r)
    d = np.cross(f, r)
    R = np.stack([r, d, f])
    t = -R @ np.asarray(c, float)
    return np.concatenate([R, t[:, None]], axis=1)


def rodrigues(axis: np.ndarray, angle: float) -> np.ndarray:
    a = np.asarray(axis, float)
    a = a / np.linalg.norm(a)
    Kx = np.array([[0, -a[2], a[1]], [a[2], 0, -a[0]], [-a[1], a[0], 0]])
    return np.eye(3) + math.sin(angle) * Kx + (1 - math.cos(angle)) * (Kx @ Kx)


def camera_centres(poses: np.ndarray) -> np.ndarray:
    P = poses.reshape(-1, 3, 4)
    return -np.einsum("nji,nj->ni", P[:, :, :3], P[:, :, 3])


def perturb_poses(rng: SplitMix64, poses: np.ndarray, angle_deg: float, frac: float,
                  pairs: np.ndarray) -> np.ndarray:
    """Initial pose = GT with the rotation perturbed by `angle_deg` about a uniform random axis and the
    camera centre moved by `frac` x (mean pair baseline) in a uniform random direction."""
    P = poses.reshape(-1, 3, 4)
    n = P.shape[0]
    C = camera_centres(poses)
    base = float(np.mean(np.linalg.norm(C[pairs[:, 0]] - C[pairs[:, 1]], axis=1)))
    axes = rng.unit_vectors(n)
    dirs = rng.unit_vectors(n)
    out = np.empty_like(P)
    for i in range(n):
        R = rodrigues(axes[i], math.radians(angle_deg)) @ P[i, :, :3]
        c = C[i] + frac * base * dirs[i]
        out[i, :, :3] = R
        out[i, :, 3] = -R @ c
    return out.reshape(n, 12)


def all_directed_pairs(n: int) -> np.ndarray:
    s, t = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
    m = s != t
    return np.stack([s[m], t[m]], axis=1).astype(np.int32)


def knn_pairs(centres: np.ndarray, k: int) -> np.ndarray:
    """Each view -> its k nearest views by camera-centre distance (ties -> lower index)."""
    n = centres.shape[0]
    d = np.linalg.norm(centres[:, None, :] - centres[None, :, :], axis=2)
    np.fill_diagonal(d, np.inf)
    out = []
    for i in range(n):
        order = np.lexsort((np.arange(n), d[i]))[:k]
        out.extend((i, int(j)) for j in order)
    return np.asarray(out, dtype=np.int32)


# ------------------------------------------------------------------------------------------------
# geometry: room (6 planes) and orbit scene (ground + boxes)
# ------------------------------------------------------------------------------------------------
ROOM = np.array([4.0, 4.0, 3.0])


def room_segments(rng: SplitMix64, count: int, len_lo: float, len_hi: float, margin: float = 0.2):
    """`count` 3-D segments on the six faces of the room [0,4]x[0,4]x[0,3]: face chosen in proportion
    to its area, first endpoint uniform inside the margin, in-plane direction uniform, length
    U(len_lo, len_hi), rejected if the second endpoint leaves the margin."""
    faces = []  # (fixed axis, value, (a, b) free axes)
    for ax in range(3):
        a, b = [i for i in range(3) if i != ax]
        for val in (0.0, ROOM[ax]):
            faces.append((ax, val, a, b, ROOM[a] * ROOM[b]))
    areas = np.array([f[4] for f in faces])
    cdf = np.cumsum(areas) / areas.sum()
    segs = []
    while len(segs) < count:
        u = rng.uniform(5)
        ax, val, a, b, _ = faces[int(np.searchsorted(cdf, u[0], side="right").clip(0, 5))]
        p0 = np.array([margin + u[1] * (ROOM[a] - 2 * margin), margin + u[2] * (ROOM[b] - 2 * margin)])
        ang = 2 * math.pi * u[3]
        ln = len_lo + (len_hi - len_lo) * u[4]
        p1 = p0 + ln * np.array([math.cos(ang), math.sin(ang)])
        if not (margin <= p1[0] <= ROOM[a] - margin and margin <= p1[1] <= ROOM[b] - margin):
            continue
        A = np.zeros(3); B = np.zeros(3)
        A[ax] = val; B[ax] = val
        A[a], A[b] = p0
        B[a], B[b] = p1
        segs.append((A, B))
    return np.asarray(segs)  # [S,2,3]


def render_depth_room(K, pose, W, H):
    """z-depth of the room's walls seen from inside, by closed-form ray/plane intersection."""
    fx, fy, cx, cy = [float(x) for x in K]
    R = pose[:, :3]; c = -R.T @ pose[:, 3]
    u = (np.arange(W) - cx) / fx
    v = (np.arange(H) - cy) / fy
    dc = np.stack(np.broadcast_arrays(u[None, :], v[:, None], np.ones((H, W))), axis=-1)  # [H,W,3]
    dw = dc @ R  # R^T d_c, row-vector form
    t = np.full((H, W), np.inf)
    for ax in range(3):
        d = dw[..., ax]
        with np.errstate(divide="ignore", invalid="ignore"):
            tp = np.where(d > 1e-12, (ROOM[ax] - c[ax]) / d, np.inf)
            tn = np.where(d < -1e-12, (0.0 - c[ax]) / d, np.inf)
        t = np.minimum(t, np.minimum(tp, tn))
    return t  # camera-frame ray has z = 1, so the ray parameter IS the z-depth


def orbit_geometry(rng: SplitMix64, n_boxes: int, count: int, area: float = 10.0, seg_scale: float = 1.0):
    """Ground plane z=0 plus `n_boxes` axis-aligned boxes inside an area x area patch; `count` segments:
    the 12 edges of every box, then random segments on the ground (length seg_scale x U(0.5, 2.5)) and on
    box faces (two uniform points, the second pulled towards the first by seg_scale)."""
    u = rng.uniform(5 * n_boxes).reshape(n_boxes, 5)
    sx = 0.3 + 0.9 * u[:, 0]; sy = 0.3 + 0.9 * u[:, 1]; h = 0.3 + 1.7 * u[:, 2]
    x0 = u[:, 3] * (area - sx); y0 = u[:, 4] * (area - sy)
    boxes = np.stack([x0, y0, np.zeros(n_boxes), x0 + sx, y0 + sy, h], axis=1)  # lo xyz, hi xyz
    segs = []
    for b in boxes:
        lo, hi = b[:3], b[3:]
        cs = np.array([[lo[0], lo[1]], [hi[0], lo[1]], [hi[0], hi[1]], [lo[0], hi[1]]])
        for k in range(4):
            a2, b2 = cs[k], cs[(k + 1) % 4]
            segs.append(([a2[0], a2[1], lo[2]], [b2[0], b2[1], lo[2]]))
            segs.append(([a2[0], a2[1], hi[2]], [b2[0], b2[1], hi[2]]))
            segs.append(([a2[0], a2[1], lo[2]], [a2[0], a2[1], hi[2]]))
    segs = segs[:count]
    # faces of boxes: 4 sides + top, chosen in proportion to area; ground chosen half of the time
    faces = []
    for b in boxes:
        lo, hi = b[:3], b[3:]
        faces.append((2, hi[2], (lo[0], hi[0]), (lo[1], hi[1])))          # top: z fixed, x-y free
        for val in (lo[0], hi[0]):
            faces.append((0, val, (lo[1], hi[1]), (lo[2], hi[2])))       # x fixed, y-z free
        for val in (lo[1], hi[1]):
            faces.append((1, val, (lo[0], hi[0]), (lo[2], hi[2])))       # y fixed, x-z free
    farea = np.array([(f[2][1] - f[2][0]) * (f[3][1] - f[3][0]) for f in faces])
    cdf = np.cumsum(farea) / farea.sum()
    while len(segs) < count:
        r = rng.uniform(6)
        if r[0] < 0.5:  # ground segment, length U(0.5, 2.5), kept inside the patch
            p0 = r[1:3] * area
            ang = 2 * math.pi * r[3]
            p1 = p0 + seg_scale * (0.5 + 2.0 * r[4]) * np.array([math.cos(ang), math.sin(ang)])
            if not (0 <= p1[0] <= area and 0 <= p1[1] <= area):
                continue
            segs.append(([p0[0], p0[1], 0.0], [p1[0], p1[1], 0.0]))
        else:           # two uniform points on a box face
            ax, val, ra, rb = faces[int(np.searchsorted(cdf, r[1], side="right").clip(0, len(faces) - 1))]
            fa, fb = [i for i in range(3) if i != ax]
            A = np.zeros(3); B = np.zeros(3)
            A[ax] = val; B[ax] = val
            A[fa] = ra[0] + r[2] * (ra[1] - ra[0]); A[fb] = rb[0] + r[3] * (rb[1] - rb[0])
            B[fa] = ra[0] + r[4] * (ra[1] - ra[0]); B[fb] = rb[0] + r[5] * (rb[1] - rb[0])
            segs.append((A, A + seg_scale * (B - A)))
    return boxes, np.asarray(segs, dtype=float)


def render_depth_orbit(K, pose, W, H, boxes, far: float = 50.0):
    """z-depth of ground plane + boxes; rays that hit nothing within `far` get depth 0."""
    fx, fy, cx, cy = [float(x) for x in K]
    R = pose[:, :3]; tvec = pose[:, 3]; c = -R.T @ tvec
    u = (np.arange(W) - cx) / fx
    v = (np.arange(H) - cy) / fy
    dc = np.stack(np.broadcast_arrays(u[None, :], v[:, None], np.ones((H, W))), axis=-1)
    dw = dc @ R
    with np.errstate(divide="ignore", invalid="ignore"):
        t = np.where(dw[..., 2] < -1e-12, -c[2] / dw[..., 2], np.inf)
    for b in boxes:
        lo, hi = b[:3], b[3:]
        corners = np.array([[x, y, z] for x in (lo[0], hi[0]) for y in (lo[1], hi[1]) for z in (lo[2], hi[2])])
        pc = corners @ R.T + tvec
        if np.all(pc[:, 2] > 0.05):
            px = fx * pc[:, 0] / pc[:, 2] + cx; py = fy * pc[:, 1] / pc[:, 2] + cy
            u0 = int(max(0, math.floor(px.min()) - 1)); u1 = int(min(W, math.ceil(px.max()) + 2))
            v0 = int(max(0, math.floor(py.min()) - 1)); v1 = int(min(H, math.ceil(py.max()) + 2))
            if u0 >= u1 or v0 >= v1:
                continue
        else:
            u0, u1, v0, v1 = 0, W, 0, H
        d = dw[v0:v1, u0:u1]
        tmin = np.zeros(d.shape[:2]); tmax = np.full(d.shape[:2], np.inf)
        for ax in range(3):
            with np.errstate(divide="ignore", invalid="ignore"):
                inv = 1.0 / d[..., ax]
                ta = (lo[ax] - c[ax]) * inv; tb = (hi[ax] - c[ax]) * inv
            tn = np.minimum(ta, tb); tf = np.maximum(ta, tb)
            par = np.abs(d[..., ax]) < 1e-12
            inside = (lo[ax] <= c[ax] <= hi[ax])
            tn = np.where(par, -np.inf if inside else np.inf, tn)
            tf = np.where(par, np.inf if inside else -np.inf, tf)
            tmin = np.maximum(tmin, tn); tmax = np.minimum(tmax, tf)
        hit = (tmin <= tmax) & (tmin > 0)
        sub = t[v0:v1, u0:u1]
        t[v0:v1, u0:u1] = np.where(hit & (tmin < sub), tmin, sub)
    return np.where(np.isfinite(t) & (t < far), t, 0.0)


# ------------------------------------------------------------------------------------------------
# edge masks
# ------------------------------------------------------------------------------------------------
def rasterize_segments(K, pose, W, H, segs, depth_gt: Optional[np.ndarray], halfwidth: float = 0.5,
                       vis_tol: float = 0.01, z_clip: float = 0.05) -> np.ndarray:
    """Mask of pixels whose centre lies within `halfwidth` px of a projected segment (clipped at
    z = z_clip) and, when `depth_gt` is given, where the segment point nearest to the pixel has a depth
    within `vis_tol` (relative) of the rendered depth there (visibility)."""
    fx, fy, cx, cy = [float(x) for x in K]
    R = pose[:, :3]; tvec = pose[:, 3]
    A = segs[:, 0] @ R.T + tvec; B = segs[:, 1] @ R.T + tvec
    za, zb = A[:, 2], B[:, 2]
    keep = (za > z_clip) | (zb > z_clip)
    A, B, za, zb = A[keep], B[keep], za[keep], zb[keep]
    # clip the endpoint that is behind z_clip
    with np.errstate(divide="ignore", invalid="ignore"):
        sa = np.where(za < z_clip, (z_clip - za) / (zb - za), 0.0)
        sb = np.where(zb < z_clip, (z_clip - zb) / (za - zb), 0.0)
    A2 = A + sa[:, None] * (B - A); B2 = B + sb[:, None] * (A - B)
    A, B = A2, B2
    a = np.stack([fx * A[:, 0] / A[:, 2] + cx, fy * A[:, 1] / A[:, 2] + cy], axis=1)
    b = np.stack([fx * B[:, 0] / B[:, 2] + cx, fy * B[:, 1] / B[:, 2] + cy], axis=1)
    iza, izb = 1.0 / A[:, 2], 1.0 / B[:, 2]
    # Liang-Barsky clip of the 2-D segment to the image rectangle grown by the half-width
    pad = halfwidth + 1.0
    lo = np.array([-pad, -pad]); hi = np.array([W - 1 + pad, H - 1 + pad])
    dlt = b - a
    s0 = np.zeros(len(a)); s1 = np.ones(len(a)); ok = np.ones(len(a), bool)
    for ax in range(2):
        d = dlt[:, ax]
        with np.errstate(divide="ignore", invalid="ignore"):
            t_lo = (lo[ax] - a[:, ax]) / d; t_hi = (hi[ax] - a[:, ax]) / d
        ent = np.where(d > 0, t_lo, t_hi); ext = np.where(d > 0, t_hi, t_lo)
        par = np.abs(d) < 1e-12
        ok &= ~(par & ((a[:, ax] < lo[ax]) | (a[:, ax] > hi[ax])))
        ent = np.where(par, -np.inf, ent); ext = np.where(par, np.inf, ext)
        s0 = np.maximum(s0, ent); s1 = np.minimum(s1, ext)
    ok &= s0 <= s1
    a, b, dlt, iza, izb, s0, s1 = a[ok], b[ok], dlt[ok], iza[ok], izb[ok], s0[ok], s1[ok]
    mask = np.zeros((H, W), np.uint8)
    if len(a) == 0:
        return mask
    pa = a + s0[:, None] * dlt; pb = a + s1[:, None] * dlt           # clipped part that is marched
    major = (np.abs(dlt[:, 1]) > np.abs(dlt[:, 0])).astype(int)       # 0: x-major, 1: y-major
    idx = np.arange(len(a))
    ma, mb = pa[idx, major], pb[idx, major]
    gpad = int(math.ceil(halfwidth)) + 1
    m_lo = np.floor(np.minimum(ma, mb)).astype(np.int64) - gpad
    m_hi = np.ceil(np.maximum(ma, mb)).astype(np.int64) + gpad
    L = (m_hi - m_lo + 1)
    seg = np.repeat(idx, L)
    off = np.arange(L.sum()) - np.repeat(np.cumsum(L) - L, L)
    m = (m_lo[seg] + off).astype(float)                                # major coordinate of each step
    dmaj = dlt[seg, major[seg]]; dmin = dlt[seg, 1 - major[seg]]
    with np.errstate(divide="ignore", invalid="ignore"):
        slope = np.where(np.abs(dmaj) > 1e-12, dmin / dmaj, 0.0)
    mclamp = np.clip(m, np.minimum(ma, mb)[seg], np.maximum(ma, mb)[seg])
    centre = a[seg, 1 - major[seg]] + slope * (mclamp - a[seg, major[seg]])
    kk = int(math.ceil(halfwidth * math.sqrt(2.0))) + 1
    ks = np.arange(-kk, kk + 1)
    mn = np.round(centre)[:, None] + ks[None, :]                        # [T, 2kk+1] minor coordinate
    mj = np.broadcast_to(m[:, None], mn.shape)
    segb = np.broadcast_to(seg[:, None], mn.shape)
    isx = (major[segb] == 0)
    px = np.where(isx, mj, mn); py = np.where(isx, mn, mj)
    px = px.ravel(); py = py.ravel(); sg = segb.ravel()
    inb = (px >= 0) & (px <= W - 1) & (py >= 0) & (py <= H - 1)
    px, py, sg = px[inb], py[inb], sg[inb]
    # exact point-to-segment distance (to the full, unclipped 2-D segment) and closest-point parameter
    ax_, ay_ = a[sg, 0], a[sg, 1]
    dx, dy = dlt[sg, 0], dlt[sg, 1]
    l2 = dx * dx + dy * dy
    with np.errstate(divide="ignore", invalid="ignore"):
        s = np.where(l2 > 1e-18, ((px - ax_) * dx + (py - ay_) * dy) / l2, 0.0)
    s = np.clip(s, 0.0, 1.0)
    qx = ax_ + s * dx; qy = ay_ + s * dy
    near = (px - qx) ** 2 + (py - qy) ** 2 <= halfwidth * halfwidth
    px, py, sg, s = px[near].astype(np.int64), py[near].astype(np.int64), sg[near], s[near]
    if depth_gt is not None:
        zseg = 1.0 / ((1.0 - s) * iza[sg] + s * izb[sg])                # perspective-correct depth
        D = depth_gt[py, px]
        vis = (D > 0) & (np.abs(zseg - D) <= vis_tol * D)
        px, py = px[vis], py[vis]
    mask[py, px] = 1
    return mask


# ------------------------------------------------------------------------------------------------
# the five BASELINE.json configurations
# ------------------------------------------------------------------------------------------------
CONFIGS = {
    1: dict(name="tiny", kind="room", N=4, W=128, H=96, f=110.0, segments=60, seg_len=(0.3, 1.5),
            layout="arc", pairs="all", depth_noise=0.0, outliers=0.0, spurious=0.0,
            init_deg=2.0, init_frac=0.05, iters=200, early_stop=0, dtf_format=0),
    2: dict(name="room24", kind="room", N=24, W=518, H=392, f=450.0, segments=400, seg_len=(0.5, 2.3),
            layout="forward", pairs="all", depth_noise=0.01, outliers=0.0, spurious=0.0,
            init_deg=3.0, init_frac=0.05, iters=200, early_stop=0, dtf_format=0),
    3: dict(name="orbit100", kind="orbit", N=100, W=518, H=392, f=450.0, segments=1500, boxes=30,
            layout="orbit", pairs=("knn", 10), depth_noise=0.02, outliers=0.01, spurious=0.05,
            init_deg=3.0, init_frac=0.05, iters=200, early_stop=0, dtf_format=0),
    4: dict(name="room200", kind="room", N=200, W=518, H=294, f=450.0, segments=400, seg_len=(0.5, 2.3),
            layout="forward", pairs="all", depth_noise=0.01, outliers=0.0, spurious=0.0,
            init_deg=2.0, init_frac=0.03, iters=200, early_stop=0, dtf_format=0),
    5: dict(name="orbit500", kind="orbit", N=500, W=518, H=392, f=450.0, segments=4000, boxes=30, seg_scale=0.35,
            layout="orbit", pairs=("knn", 20), depth_noise=0.02, outliers=0.02, spurious=0.0,
            init_deg=5.0, init_frac=0.10, iters=2000, early_stop=1, dtf_format=0),
}


def _cameras(rng: SplitMix64, cfg: dict) -> np.ndarray:
    n = cfg["N"]
    poses = np.empty((n, 3, 4))
    if cfg["layout"] == "arc":          # 60-degree arc of radius 1.4 around the box centre, looking inward
        centre = ROOM / 2
        dz = rng.uniform(n, -0.3, 0.3)
        for i in range(n):
            a = math.radians(-30.0 + 60.0 * i / max(n - 1, 1))
            c = centre + np.array([-1.4 * math.cos(a), 1.4 * math.sin(a), dz[i]])
            poses[i] = look_at(c, centre)
    elif cfg["layout"] == "forward":    # forward-facing: centres in a slab, looking at a far-wall patch
        u = rng.uniform(6 * n).reshape(n, 6)
        for i in range(n):
            c = np.array([0.4 + 1.2 * u[i, 0], 0.8 + 2.4 * u[i, 1], 1.0 + 1.0 * u[i, 2]])
            tgt = np.array([4.0, 1.2 + 1.6 * u[i, 3], 1.0 + 1.0 * u[i, 4]])
            poses[i] = look_at(c, tgt)
    elif cfg["layout"] == "orbit":      # circle of radius 9 around the scene centre, height U(1.5, 3)
        u = rng.uniform(4 * n).reshape(n, 4)
        for i in range(n):
            a = 2 * math.pi * i / n
            c = np.array([5.0 + 9.0 * math.cos(a), 5.0 + 9.0 * math.sin(a), 1.5 + 1.5 * u[i, 0]])
            tgt = np.array([5.0, 5.0, 0.5]) + (u[i, 1:4] - 0.5) * 0.6
            poses[i] = look_at(c, tgt)
    else:
        raise ValueError(cfg["layout"])
    return poses


def make_scene(config: int, *, n_views: Optional[int] = None, seed: Optional[int] = None,
               overrides: Optional[dict] = None, target_halfwidth: Optional[float] = None) -> Scene:
    """Build BASELINE.json config `config` (1..5).  `n_views` / `overrides` shrink or alter it for tests
    (same generator, same statistics).  `target_halfwidth` rasterises the masks as bands of that
    half-width instead of 0.5 px (used by the exact-zero-loss pin)."""
    cfg = dict(CONFIGS[config])
    if overrides:
        cfg.update(overrides)
    if n_views is not None:
        cfg["N"] = n_views
    root = SplitMix64(BASE_SEED + config if seed is None else seed)
    r_geo, r_cam, r_init, r_noise = root.fork(1), root.fork(2), root.fork(3), root.fork(4)
    W, H, n = cfg["W"], cfg["H"], cfg["N"]
    K = np.tile(np.array([cfg["f"], cfg["f"], W / 2.0, H / 2.0]), (n, 1))
    if cfg["kind"] == "room":
        segs = room_segments(r_geo, cfg["segments"], *cfg["seg_len"]); boxes = None
    else:
        boxes, segs = orbit_geometry(r_geo, cfg["boxes"], cfg["segments"], seg_scale=cfg.get("seg_scale", 1.0))
    poses = _cameras(r_cam, cfg)
    depth = np.empty((n, H, W), np.float32); edges = np.empty((n, H, W), np.uint8)
    hw = 0.5 if target_halfwidth is None else target_halfwidth
    for i in range(n):
        d = render_depth_room(K[i], poses[i], W, H) if boxes is None else \
            render_depth_orbit(K[i], poses[i], W, H, boxes)
        # band masks (Z0 pin) skip the 1 % visibility test: a band pixel 3 px off a segment on a steep wall
        # differs in depth by more than that; the room is convex, so nothing is occluded anyway
        m = rasterize_segments(K[i], poses[i], W, H, segs, d if target_halfwidth is None else None, halfwidth=hw)
        rn = r_noise.fork(i)
        if cfg["spurious"] > 0:                       # A4: 5 % of the view's true edge count, uniform positions
            k = int(round(cfg["spurious"] * int(m.sum())))
            pu = rn.integers(k, W); pv = rn.integers(k, H)
            m[pv, pu] = 1
        if cfg["depth_noise"] > 0:
            d = d * (1.0 + cfg["depth_noise"] * rn.normal(H * W).reshape(H, W))
        if cfg["outliers"] > 0:
            sel = rn.uniform(H * W).reshape(H, W) < cfg["outliers"]
            d = np.where(sel, rn.uniform(H * W, 0.5, 2.0 * float(d.max())).reshape(H, W), d)
        depth[i] = d.astype(np.float32); edges[i] = m
    poses_gt = poses.reshape(n, 12)
    if cfg["pairs"] == "all":
        pairs = all_directed_pairs(n)
    else:
        pairs = None
    # initial poses; the kNN list is drawn from the INITIAL centres (what a 3DFM front-end would supply)
    base_pairs = pairs if pairs is not None else knn_pairs(camera_centres(poses_gt), min(cfg["pairs"][1], n - 1))
    poses_init = perturb_poses(r_init, poses_gt, cfg["init_deg"], cfg["init_frac"], base_pairs)
    if pairs is None:
        pairs = knn_pairs(camera_centres(poses_init.astype(np.float32).astype(np.float64)),
                          min(cfg["pairs"][1], n - 1))
    meta = dict(cfg); meta["config"] = config; meta["seed"] = int(root.seed)
    return Scene(name=cfg["name"], W=W, H=H, K=K.astype(np.float32), poses_gt=poses_gt,
                 poses_init=poses_init.astype(np.float32), depth=depth, edges=edges,
                 pairs=np.ascontiguousarray(pairs, dtype=np.int32), meta=meta)
