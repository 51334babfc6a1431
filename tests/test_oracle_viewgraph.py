"""Pins of the oracle's viewgraph estimation by cycle-consistent reprojection (Eq. 2, 117, 380-384,
396): closed forms on fronto-parallel planes, degenerate geometries, the 12.5 % / both-directions rule on hand-made
counts, and the rendered room at ground truth.  No value here comes from the routine under test."""
import numpy as np

import oracle
from epo_scenes import make_scene

W, H, F = 160, 120, 100.0


def _cams(T_list):
    K = np.tile(np.array([F, F, W / 2, H / 2], np.float32), (len(T_list), 1))
    return K, np.stack(T_list).astype(np.float64).reshape(len(T_list), 12)


def _eye(tx=0.0, ry_deg=0.0):
    c, s = np.cos(np.radians(ry_deg)), np.sin(np.radians(ry_deg))
    T = np.array([[c, 0, s, tx], [0, 1, 0, 0], [-s, 0, c, 0]], np.float64)
    return T


def _grid_u(stride):
    return np.arange(stride // 2, W, stride), np.arange(stride // 2, H, stride)


def test_V1_identical_cameras_keep_every_usable_point():
    K, P = _cams([_eye(), _eye()])
    depth = np.full((2, H, W), 5.0, np.float32)
    depth[0, :, :40] = 0.0                                   # unusable depth: not counted at all (reading V2)
    depth[0, 60, 100] = np.inf
    for fp32 in (0, 1):
        c = oracle.viewgraph_counts(K, P, depth, stride=8, tau=3.0, coord_fp32=fp32)
        us, vs = _grid_u(8)
        usable0 = sum(1 for v in vs for u in us if u >= 40 and not (v == 60 and u == 100))
        assert tuple(c[0, 1]) == (usable0, usable0)
        # from view 1 every grid point is usable but those landing on view 0's holes find no depth there
        assert c[1, 0, 1] == len(us) * len(vs) and c[1, 0, 0] == usable0
        assert tuple(c[0, 0]) == (0, 0) and tuple(c[1, 1]) == (0, 0)


def test_V2_closed_form_translation_and_the_strict_threshold():
    """Fronto-parallel plane at Z0 seen by two cameras b apart along x: p lands at u - F b / Z0; if view j's depth map
    says Z' instead of Z0 the round trip misses by e = F b |1/Z' - 1/Z0| exactly.  e = 2.9 px keeps the point,
    e = 3.1 px drops it (tau = 3, strict <)."""
    b, Z0 = 1.0, 10.0
    K, P = _cams([_eye(), _eye(tx=-b)])                      # camera 1 centre at x = +b
    us, vs = _grid_u(8)
    lands = sum(1 for v in vs for u in us if u - F * b / Z0 >= 0.0)      # shift of 10 px to the left
    for e, keep in ((0.0, True), (2.9, True), (3.1, False)):
        Zp = 1.0 / (1.0 / Z0 - e / (F * b))
        depth = np.stack([np.full((H, W), Z0, np.float32), np.full((H, W), Zp, np.float32)])
        for fp32 in (0, 1):
            c = oracle.viewgraph_counts(K, P, depth, stride=8, tau=3.0, coord_fp32=fp32)
            assert c[0, 1, 1] == len(us) * len(vs)
            assert c[0, 1, 0] == (lands if keep else 0), (e, fp32, c[0, 1])


def test_V3_opposite_cameras_share_nothing_and_are_rejected():
    K, P = _cams([_eye(), _eye(ry_deg=180.0)])
    depth = np.full((2, H, W), 4.0, np.float32)
    c = oracle.viewgraph_counts(K, P, depth)
    assert c[0, 1, 0] == 0 and c[1, 0, 0] == 0 and c[0, 1, 1] > 0
    assert len(oracle.viewgraph_pairs(c)) == 0


def test_V4_pair_rule_on_hand_made_counts():
    """>= 12.5 % in BOTH directions (reading V7); usable = 0 rejects; pairs come as (i,j),(j,i), i<j ascending."""
    c = np.zeros((4, 4, 2), np.int32)
    c[0, 1] = (1, 8); c[1, 0] = (2, 8)        # exactly 12.5 % and above: kept
    c[0, 2] = (1, 9); c[2, 0] = (9, 9)        # 11.1 % one way: rejected
    c[1, 3] = (5, 5); c[3, 1] = (0, 0)        # nothing usable on the way back: rejected
    c[2, 3] = (100, 800); c[3, 2] = (700, 800)
    assert oracle.viewgraph_pairs(c).tolist() == [[0, 1], [1, 0], [2, 3], [3, 2]]
    assert oracle.viewgraph_pairs(c, min_frac=0.2).tolist() == []
    assert oracle.viewgraph_pairs(c, min_frac=0.5).tolist() == []
    assert oracle.viewgraph_pairs(c, min_frac=0.1).tolist() == [[0, 1], [1, 0], [0, 2], [2, 0], [2, 3], [3, 2]]


def test_V5_rendered_room_at_ground_truth_and_under_a_wrong_pose():
    """Noise-free rendered depth at GT poses: a cycle can only fail through occlusion / leaving the image / the
    nearest-pixel depth across a wall corner, so overlapping forward-facing views keep most points; turning one camera
    by 70 degrees breaks its cycles with everyone."""
    sc = make_scene(2, n_views=5, overrides=dict(depth_noise=0.0))
    c = oracle.viewgraph_counts(sc.K, sc.poses_gt, sc.depth, stride=8, tau=3.0)
    frac = c[..., 0] / np.maximum(c[..., 1], 1)
    off = ~np.eye(5, dtype=bool)
    assert frac[off].min() > 0.3 and np.median(frac[off]) > 0.5
    assert len(oracle.viewgraph_pairs(c)) == 20
    bad = sc.poses_gt.astype(np.float64).reshape(5, 3, 4).copy()
    a = np.radians(70.0); R = np.array([[np.cos(a), 0, np.sin(a)], [0, 1, 0], [-np.sin(a), 0, np.cos(a)]])
    bad[2] = R @ bad[2]
    cb = oracle.viewgraph_counts(sc.K, bad.reshape(5, 12), sc.depth, stride=8, tau=3.0)
    fb = cb[..., 0] / np.maximum(cb[..., 1], 1)
    assert fb[2, [0, 1, 3, 4]].max() < 0.02 and fb[[0, 1, 3, 4], 2].max() < 0.02
    others = [[i, j] for i in (0, 1, 3, 4) for j in (0, 1, 3, 4) if i != j]
    assert sorted(oracle.viewgraph_pairs(cb).tolist()) == sorted(others)
    # the binary32-position variant takes the same decisions up to a few borderline grid points
    c32 = oracle.viewgraph_counts(sc.K, sc.poses_gt, sc.depth, stride=8, tau=3.0, coord_fp32=1)
    assert np.abs(c32 - c).max() <= 3 and np.array_equal(c32[..., 1], c[..., 1])


def test_V6_uncertain_counts_bound_a_binary32_evaluation():
    """orc_viewgraph_counts_slack (reading T1): its (consistent, usable) ARE the all-double counts; the
    binary32-position variant -- one concrete binary32 evaluation -- differs from them by at most the `uncertain` count
    of the pair, on scenes where it does differ; the uncertain points are a small minority; and the pairs that are
    valid whatever the uncertain points decide are a subset of the binary32 variant's list, which is a subset of the
    pairs valid for some decision."""
    differed = 0
    for cfg, nv, stride in ((1, None, 4), (2, 6, 8), (3, 8, 8), (5, 10, 5)):
        sc = make_scene(cfg, n_views=nv)
        poses = sc.poses_init.astype(np.float64)
        c3 = oracle.viewgraph_counts_slack(sc.K, poses, sc.depth, stride=stride, tau=3.0)
        c64 = oracle.viewgraph_counts(sc.K, poses, sc.depth, stride=stride, tau=3.0)
        c32 = oracle.viewgraph_counts(sc.K, poses, sc.depth, stride=stride, tau=3.0, coord_fp32=1)
        assert np.array_equal(c3[..., :2], c64)
        assert np.array_equal(c32[..., 1], c64[..., 1])
        assert np.all(np.abs(c32[..., 0] - c64[..., 0]) <= c3[..., 2])
        differed += int(np.sum(c32[..., 0] != c64[..., 0]))
        assert c3[..., 2].sum() <= 0.02 * c3[..., 1].sum()
        certain, possible = oracle.viewgraph_pairs_robust(c3, 0.125)
        got = np.zeros_like(certain)
        for i, j in oracle.viewgraph_pairs(c32, 0.125):
            if i < j: got[i, j] = True
        assert np.all(got[certain]) and not np.any(got & ~possible)
    assert differed >= 1
