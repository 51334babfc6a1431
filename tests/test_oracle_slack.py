"""Pins for the oracle's event slack (orc_pair_event_slack / orc_event_slack, reading T1): the bound on
what a correct binary32 evaluation of the loss may decide differently from the all-double oracle.

T1a  the slack routine's own per-sample terms, summed over the nominal decisions, ARE the pinned pair routine's sums
T1b  closed forms: a sample exactly on the clamp boundary d = lambda, and a sample exactly on a bilinear-cell border
     where the field has a kink with d != 0 -- the slack is the hand-computed jump, everything else contributes none
T1c  the bound holds: the all-double loss re-evaluated with every projected position displaced by less than the
     stated binary32 position error (principal point of the target shifted by +-delta px) stays within
     1e-6 relative + slack of the nominal result, pair by pair, on a scene where such displacements do flip samples;
     and the oracle's binary32-position variant (one concrete binary32 evaluation) stays within it too
T1d  the bound is not vacuous on a realistic scene (a few 1e-3 of the gradient norm), and is zero without events
"""
import numpy as np

import oracle
from epo_scenes import make_scene


def _pair_inputs(sc, prob, s, t):
    lo, hi = prob.edge_off[s], prob.edge_off[s + 1]
    return prob.uv[lo:hi], prob.z[lo:hi], sc.K[s].astype(np.float64), sc.K[t].astype(np.float64)


def test_T1a_slack_routine_reproduces_the_pinned_sums():
    sc = make_scene(2, n_views=4)
    prob = oracle.preprocess(sc.K, sc.depth, sc.edges)
    poses = sc.poses_init.astype(np.float64)
    for s, t in sc.pairs:
        uv, z, Ks, Kt = _pair_inputs(sc, prob, s, t)
        S, nv, G, _ = oracle.pair_loss_grad(uv, z, Ks, Kt, poses[s], poses[t], prob.dtf[t], 8.0)
        chk = oracle.pair_event_slack(uv, z, Ks, Kt, poses[s], poses[t], prob.dtf[t], 8.0)["check"]
        assert chk[1] == nv and nv > 100
        assert abs(chk[0] - S) <= 1e-12 * S
        assert np.linalg.norm(chk[2:] - G) <= 1e-12 * np.linalg.norm(G)


def _fronto(W, H, cols, fx, fy, cx, cy, b, Z0, rows, by=0.0):
    m = np.zeros((H, W), np.uint8)
    for c in cols:
        m[:, c] = 1
    dtf = oracle.edt(m)
    us, vs = np.meshgrid(np.arange(W), np.asarray(rows)); us = us.ravel(); vs = vs.ravel()
    uv = np.stack([us, vs], axis=1).astype(np.uint16); z = np.full(len(us), Z0, np.float32)
    K = np.array([fx, fy, cx, cy]); Ts = np.eye(4)[:3].reshape(12); Tt = np.eye(4)[:3].copy(); Tt[0, 3] = b; Tt[1, 3] = by
    return dtf, uv, z, K, Ts, Tt.reshape(12), us, vs


def test_T1b_closed_form_clamp_boundary():
    """One edge column c: DTF = |x - c|.  x(u) = u + fx b / Z0 = u + 2.5 exactly, so no sample is near a cell border
    and exactly two samples per row sit ON d = lambda = 6.5; each may lose its whole gradient term
    a = rho' sign fx / Z0 (1, 0, -X / Z0), [a ; x_t x a], and nothing else is uncertain."""
    W, H, fx, fy, cx, cy, c, Z0, b = 96, 40, 64.0, 64.0, 47.5, 20.25, 41, 2.0, 0.078125     # 64 b / 2 = 2.5
    rows = [5, 12, 30]
    dtf, uv, z, K, Ts, Tt, us, vs = _fronto(W, H, [c], fx, fy, cx, cy, b, Z0, rows, by=0.015625)   # y = v + 0.5
    out = oracle.pair_event_slack(uv, z, K, K, Ts, Tt, dtf, 6.5, 1.0)
    x = us + 2.5
    on = np.abs(np.abs(x - c) - 6.5) < 1e-12
    assert on.sum() == 2 * len(rows) and out["flagged"] == on.sum() and out["k_out"] == 0 and out["k_in"] == 0
    sign = np.sign(x - c)[on]; X = ((us - cx) / fx * Z0 + b)[on]; Y = ((vs - cy) / fy * Z0 + 0.015625)[on]
    a = np.stack([sign * fx / Z0, np.zeros(on.sum()), -sign * fx * X / Z0 ** 2], axis=1)         # rho' = delta = 1
    xt = np.stack([X, Y, np.full(on.sum(), Z0)], axis=1)
    g = np.concatenate([a, np.cross(xt, a)], axis=1)
    assert abs(out["E_t"] - np.linalg.norm(g, axis=1).sum()) <= 1e-12 * out["E_t"]
    assert out["E_rho"] <= 1e-12                                   # rho is continuous at the clamp
    # away from the boundary value nothing is flagged at all
    clean = oracle.pair_event_slack(uv, z, K, K, Ts, Tt, dtf, 6.25, 1.0)
    assert clean["flagged"] == 0 and clean["E_t"] == 0.0 and clean["E_s"] == 0.0


def test_T1b_closed_form_cell_border_at_a_kink():
    """Two edge columns 30 and 40: DTF = min(|x - 30|, |x - 40|) has a kink with d = 5 at x = 35.  x(u) = u + 3 exactly,
    so EVERY sample sits on a cell border; only at x = 35 do the two cells differ (slope +1 | -1): the slack is twice
    that sample's gradient term per row, and zero for all the others although they are all flagged."""
    W, H, fx, fy, cx, cy, Z0, b = 96, 40, 64.0, 60.0, 47.5, 20.25, 2.0, 0.09375                  # 64 b / 2 = 3
    rows = [7, 19]
    dtf, uv, z, K, Ts, Tt, us, vs = _fronto(W, H, [30, 40], fx, fy, cx, cy, b, Z0, rows)
    out = oracle.pair_event_slack(uv, z, K, K, Ts, Tt, dtf, 10.5, 1.0)    # no sample has d = lambda
    x = us + 3.0
    valid = x <= W - 1
    assert out["flagged"] >= valid.sum() - 2 * len(rows)          # all interior samples are on a cell border
    at = x == 35.0
    X = ((us - cx) / fx * Z0 + b)[at]; Y = ((vs - cy) / fy * Z0)[at]
    a = np.stack([np.full(at.sum(), fx / Z0), np.zeros(at.sum()), -fx * X / Z0 ** 2], axis=1)    # |slope| = 1, rho' = 1
    xt = np.stack([X, Y, np.full(at.sum(), Z0)], axis=1)
    g = np.concatenate([a, np.cross(xt, a)], axis=1)
    assert abs(out["E_t"] - 2.0 * np.linalg.norm(g, axis=1).sum()) <= 1e-12 * out["E_t"]
    # x = W - 1 exactly is ON the validity border: one sample per row may be dropped
    assert out["k_out"] == len(rows) and out["k_in"] == 0


def _bounds(ref, sl, p):
    n = float(ref["pair_valid"][p]); k_out, k_in = float(sl["k_out"]), float(sl["k_in"])
    n_lo = max(n - k_out, 1.0); kmax = max(k_out, k_in)
    Gt, Gs = np.linalg.norm(ref["pair_G"][p, :6]), np.linalg.norm(ref["pair_G"][p, 6:])
    return (sl["E_t"] / n_lo + Gt * kmax / (n * n_lo), sl["E_s"] / n_lo + Gs * kmax / (n * n_lo),
            sl["E_rho"] / n_lo + ref["pair_loss"][p] * kmax / n_lo)


def test_T1c_displaced_and_binary32_evaluations_stay_within_the_bound():
    sc = make_scene(2, n_views=5)
    prob = oracle.preprocess(sc.K, sc.depth, sc.edges)
    poses = sc.poses_init.astype(np.float64)
    lam = 8.0
    ref = oracle.loss_grad(prob, poses, sc.pairs, lam, want_pair_G=True)
    b32 = oracle.loss_grad(prob, poses, sc.pairs, lam, want_pair_G=True, coord_fp32=1)
    moved = 0; used = 0
    for p, (s, t) in enumerate(sc.pairs):
        uv, z, Ks, Kt = _pair_inputs(sc, prob, s, t)
        sl = oracle.pair_event_slack(uv, z, Ks, Kt, poses[s], poses[t], prob.dtf[t], lam)
        bt, bs, bl = _bounds(ref, sl, p)
        n = ref["pair_valid"][p]
        g0 = ref["pair_G"][p] / n
        cases = [(b32["pair_G"][p], b32["pair_valid"][p], b32["pair_loss"][p])]
        for dx, dy in ((4e-6, 0.0), (-4e-6, 4e-6), (0.0, -4e-6), (4e-6, 4e-6), (-4e-6, -4e-6)):
            Kd = Kt.copy(); Kd[2] += dx; Kd[3] += dy              # every projected position moves by exactly (dx, dy)
            S, nv, G, _ = oracle.pair_loss_grad(uv, z, Ks, Kd, poses[s], poses[t], prob.dtf[t], lam)
            cases.append((G, nv, S / nv))
        for G, nv, L in cases:
            assert n - sl["k_out"] <= nv <= n + sl["k_in"]
            et = np.linalg.norm(G[:6] / nv - g0[:6]); es = np.linalg.norm(G[6:] / nv - g0[6:])
            # 2e-5: what the displacement itself moves the continuous part by
            assert et <= 2e-5 * np.linalg.norm(g0[:6]) + bt, (p, et, bt)
            assert es <= 2e-5 * np.linalg.norm(g0[6:]) + bs, (p, es, bs)
            assert abs(L - ref["pair_loss"][p]) <= 2e-5 * ref["pair_loss"][p] + bl
            used += 1
            moved += et > 2e-5 * np.linalg.norm(g0[:6])
    # the displacements did flip samples (the test bites), and the flips stayed inside the bound
    assert moved >= 5, (moved, used)


def test_T1d_slack_is_small_where_it_should_be():
    sc = make_scene(2, n_views=5)
    prob = oracle.preprocess(sc.K, sc.depth, sc.edges)
    poses = sc.poses_init.astype(np.float64)
    ref = oracle.loss_grad(prob, poses, sc.pairs, 10.0, want_pair_G=True)
    sl = oracle.event_slack(prob, poses, sc.pairs, 10.0, ref)
    rel = sl["cam"] / np.linalg.norm(ref["grad"], axis=1)
    frac = sl["flagged"].sum() / ref["pair_valid"].sum()
    print(f"room5: slack / |g| per camera {rel}, flagged samples {100 * frac:.3f} %")
    assert np.all(np.isfinite(sl["cam"])) and rel.max() < 3e-2 and frac < 1e-2
    assert np.all(sl["pair_loss"] <= 1e-3 * ref["pair_loss"] + 1e-12)
    # the per-camera slack is the pair bounds gathered by target and source
    cam = np.zeros(sc.n_views)
    for p, (s, t) in enumerate(sc.pairs):
        uv, z, Ks, Kt = _pair_inputs(sc, prob, s, t)
        bt, bs, _ = _bounds(ref, oracle.pair_event_slack(uv, z, Ks, Kt, poses[s], poses[t], prob.dtf[t], 10.0), p)
        cam[t] += bt; cam[s] += bs
    assert np.allclose(cam / len(sc.pairs), sl["cam"], rtol=1e-12, atol=0)


def test_T1e_joint_phase_slack_holds_for_displaced_and_binary32_evaluations():
    """The same bound for the joint phase's gradients (orc_joint_slack): d L / d ln f per camera and d L / d Z per edge
    pixel of evaluations whose projected positions are displaced by less than the binary32 position error (all
    principal points shifted by a few 1e-6 px) and of the oracle's binary32-position variant stay within
    2e-5 relative + slack of the nominal all-double result; entries without any event in reach have zero slack."""
    import copy
    sc = make_scene(2, n_views=5)
    prob = oracle.preprocess(sc.K, sc.depth, sc.edges)
    poses = sc.poses_init.astype(np.float64)
    lam = 8.0
    gf, gz = oracle.joint_grad(prob, poses, sc.pairs, lam)
    sl = oracle.joint_slack(prob, poses, sc.pairs, lam)
    assert np.all(np.isfinite(sl["logf"])) and np.all(np.isfinite(sl["gz"]))
    assert (sl["gz"] == 0).mean() > 0.95 and (sl["gz"] > 0).sum() > 10
    scale_f = np.maximum(np.abs(gf), sl["logf_rss"])
    cases = [oracle.joint_grad(prob, poses, sc.pairs, lam, coord_fp32=1)]
    for dx, dy in ((3e-6, 0.0), (-3e-6, 3e-6), (3e-6, -3e-6)):
        p2 = copy.copy(prob); p2.K = prob.K.astype(np.float64)
        # float32 intrinsics cannot carry a 1e-6 px shift: displace through the (double) poses instead -- a rotation
        # of every camera about its own y / x axis by dx / fx, dy / fy moves every projection by about (dx, dy)
        P2 = poses.reshape(-1, 3, 4).copy()
        for c in range(sc.n_views):
            ax, ay = dy / sc.K[c, 1], -dx / sc.K[c, 0]
            R = np.array([[1, 0, -ay], [0, 1, ax], [ay, -ax, 1.0]])          # first order: Exp of a 1e-8 rad twist
            P2[c] = R @ P2[c]
        cases.append(oracle.joint_grad(prob, P2.reshape(-1, 12), sc.pairs, lam))
    moved = 0
    for k, (f2, z2) in enumerate(cases):
        # what the displacement itself moves the continuous part by: a binary32 position is off by up to ~1e-4 px, and a
        # single edge pixel's derivative (a sum over a handful of pairs, nothing averages) follows the interpolant's
        # curvature with it -- 1e-3 relative per entry, 1e-4 on a camera's sum; the 3e-6 px displacements: 2e-5
        rel_z, rel_f = (1e-3, 1e-4) if k == 0 else (2e-5, 2e-5)
        assert np.all(np.abs(f2 - gf) <= rel_f * scale_f + sl["logf"])
        tol = rel_z * np.abs(gz) + rel_z * 0.1 * np.abs(gz).max() + sl["gz"]
        assert np.all(np.abs(z2 - gz) <= tol), float(np.max(np.abs(z2 - gz) - tol))
        moved += int(np.sum((sl["gz"] > 0) & (np.abs(z2 - gz) > 0.2 * sl["gz"])))     # a flagged entry really flipped
    assert moved >= 1                                   # a flagged sample did change cell / branch, inside its slack
