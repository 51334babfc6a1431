"""Pins of the oracle's joint-phase gradients (Eq. 4-5: focal scale f = f0 (1 + gamma), pixel-wise depth
Z = Z0 alpha + beta; "in the subsequent joint phase, optimization is extended to include the depth maps"):
central finite differences of the LOSS FUNCTION itself (orc_loss_grad's loss, pinned by Z0-Z5), never of the gradient
routine, plus two identities."""
import copy

import numpy as np

import oracle
from epo_scenes import make_scene

LAM = 10.0


def _setup():
    sc = make_scene(1)
    prob = oracle.preprocess(sc.K, sc.depth, sc.edges, z_min=1e-6)
    return sc, prob, sc.poses_init.astype(np.float64)


def _loss(prob, poses, pairs):
    return oracle.loss_grad(prob, poses, pairs, LAM)["loss"]


def test_J1_focal_gradient_matches_finite_differences():
    sc, prob, poses = _setup()
    g_f, _ = oracle.joint_grad(prob, poses, sc.pairs, LAM)
    assert np.all(np.abs(g_f) > 1e-4)
    for c in range(sc.n_views):
        f0 = float(prob.K[c, 0]); h = 2e-5
        vals = []
        for sgn in (+1, -1):
            q = copy.copy(prob); q.K = prob.K.copy()
            q.K[c, 0] = q.K[c, 1] = np.float32(f0 * np.exp(sgn * h))
            vals.append((_loss(q, poses, sc.pairs), np.log(float(q.K[c, 0]) / f0)))     # the step actually taken (fp32 K)
        fd = (vals[0][0] - vals[1][0]) / (vals[0][1] - vals[1][1])
        assert abs(fd - g_f[c]) <= 1e-3 * abs(g_f[c]), (c, fd, g_f[c])


def test_J2_depth_gradient_matches_finite_differences():
    sc, prob, poses = _setup()
    _, g_z = oracle.joint_grad(prob, poses, sc.pairs, LAM)
    rng = np.random.default_rng(3)
    # (i) one view at a time, all its depths scaled by (1 + h): dL/dh = sum_e g_z[e] Z_e -- every entry takes part
    for c in range(sc.n_views):
        lo, hi = prob.edge_off[c], prob.edge_off[c + 1]
        h = 1e-5; vals = []
        for sgn in (+1, -1):
            q = copy.copy(prob); q.z = prob.z.copy()
            q.z[lo:hi] = (prob.z[lo:hi].astype(np.float64) * (1 + sgn * h)).astype(np.float32)
            vals.append((_loss(q, poses, sc.pairs), q.z[lo:hi].astype(np.float64) - prob.z[lo:hi]))
        # first-order prediction with the steps actually taken (fp32 depths)
        pred = float(g_z[lo:hi] @ (vals[0][1] - vals[1][1]))
        fd = vals[0][0] - vals[1][0]
        assert abs(fd - pred) <= 2e-3 * abs(pred) + 1e-12, (c, fd, pred)
    # (ii) single entries
    big = np.argsort(-np.abs(g_z))[:200]
    for e in rng.choice(big, 8, replace=False):
        h = 1e-4 * float(prob.z[e]); vals = []
        for sgn in (+1, -1):
            q = copy.copy(prob); q.z = prob.z.copy(); q.z[e] = np.float32(float(prob.z[e]) + sgn * h)
            vals.append((_loss(q, poses, sc.pairs), float(q.z[e])))
        fd = (vals[0][0] - vals[1][0]) / (vals[0][1] - vals[1][1])
        assert abs(fd - g_z[e]) <= 5e-3 * abs(g_z[e]), (e, fd, g_z[e])


def test_J3_identities():
    """Scaling the whole scene (all depths and all camera centres) by k leaves every projection unchanged:
    sum_e g_z[e] Z_e + (translation part of the pose gradient contracted with the translations) = 0; and an entry whose
    sample is invalid in every pair has zero gradient; the fp32-position variant agrees with the double one."""
    sc, prob, poses = _setup()
    g_f, g_z = oracle.joint_grad(prob, poses, sc.pairs, LAM)
    ref = oracle.loss_grad(prob, poses, sc.pairs, LAM)
    # d/dk at k = 1 of L(k Z, R, k t): world-to-camera t scales with the scene; left-perturbation gradient wrt v is dL/dt
    # for a pure translation increment (T <- [I | v] T adds v to t)
    t = poses.reshape(-1, 3, 4)[:, :, 3]
    total = float(g_z @ prob.z.astype(np.float64)) + float(np.sum(ref["grad"][:, :3] * t))
    scale = abs(float(g_z @ prob.z.astype(np.float64))) + 1e-30
    assert abs(total) <= 1e-9 * scale, (total, scale)
    g_f32, g_z32 = oracle.joint_grad(prob, poses, sc.pairs, LAM, coord_fp32=1)
    assert np.allclose(g_f32, g_f, rtol=2e-3, atol=1e-9)
    assert np.linalg.norm(g_z32 - g_z) <= 2e-2 * np.linalg.norm(g_z)
    far = make_scene(1); far.poses_init = far.poses_init.copy()
    # a view with an unusable target for everybody: push camera 3 behind the scene -> pairs into it have no valid sample
    p2 = poses.copy().reshape(-1, 3, 4); p2[3, :, 3] += np.array([0, 0, 500.0]); p2 = p2.reshape(-1, 12)
    only = np.array([[0, 3]], np.int32)
    r = oracle.loss_grad(prob, p2, only, LAM)
    if r["pair_valid"][0] == 0:
        gf, gz = oracle.joint_grad(prob, p2, only, LAM)
        assert not gf.any() and not gz.any()
