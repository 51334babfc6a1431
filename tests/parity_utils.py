"""Shared helpers of the GPU parity tests: build a library context from a Scene, and compare its outputs with
the all-double CPU oracle under BASELINE.json's tolerances.

Tolerances (BASELINE.json north_star): edge lists / pair lists / EDT bit-exact; per-pair loss 1e-5 relative;
per-camera gradient 1e-4 relative; poses after a fixed 200 iterations 1e-3 degrees and 1e-4 scene units.

The slack rule (readings T1, T2; SURVEY.md 8(c) "Tolerance realism").  The reference is ALWAYS the all-double
oracle.  Loss and gradient are continuous in the projected position except at three decisions per sample -- valid or
not, the bilinear cell, d <= lambda -- which a binary32 evaluation may take differently for the few
samples that lie within binary32 rounding of a boundary.  The oracle itself enumerates those samples and bounds what
they can move (`oracle.event_slack`, pinned by tests/test_oracle_slack.py), and every comparison here is
    | gpu - oracle | <= contract tolerance x | oracle | + slack(oracle)
with the slack reported next to the observed error; for a camera's gradient "| oracle |" is the larger of its norm
and the root-sum-square of its per-sample terms (T2: at a minimum the terms cancel and the norm alone is no scale).  The oracle's binary32-position variant (`coord_fp32=1`) is a
diagnostic only: it is printed, never asserted, and it takes part in no bound.
"""
import math

import numpy as np

Z_MIN = float(np.float32(1e-6))


def f32(x):
    return float(np.float32(x))


def oracle_config(**kw):
    """Oracle hyper-parameters equal to the library's fp32 defaults widened to double."""
    import oracle
    base = dict(huber_delta=1.0, clamp_start=10.0, clamp_end=6.0, clamp_steps=1000, lr_max=f32(3e-3),
                warmup_steps=25, max_steps=2000, beta1=f32(0.9), beta2=f32(0.999), adam_eps=f32(1e-8),
                eps1=f32(0.5), eps2=f32(0.1), w1=25, w2=50, smooth_window=1, early_stop=0, z_min=Z_MIN)
    base.update(kw)
    return oracle.Config(**base)


def make_ctx(scene, device_inputs=False, **cfg_over):
    import torch
    from paper_2607_00579_b200 import Epo, epo_config_default
    cfg = epo_config_default(n_views=scene.n_views, width=scene.W, height=scene.H,
                             stream=torch.cuda.current_stream().cuda_stream, **cfg_over)
    e = Epo(cfg)
    if device_inputs:
        t = [torch.from_numpy(a).cuda() for a in (scene.K, scene.poses_init, scene.depth, scene.edges)]
        e.set_views(*t)
        e.set_pairs(torch.from_numpy(scene.pairs).cuda())
        torch.cuda.synchronize()
    else:
        e.set_views(scene.K, scene.poses_init, scene.depth, scene.edges)
        e.set_pairs(scene.pairs)
    return e


def trajectory_spread(prob, scene, iters, o64_poses, draws, cfg_kw=None, seed=7):
    """How far apart correct evaluations of the SAME free-running loop end after `iters` iterations, measured on the
    all-double oracle alone (reading P7): the distances (degrees, scene units) from the all-double run
    `o64_poses` of `draws` all-double runs whose initial poses differ from the given ones by at most ONE ulp of binary32
    per entry (seeded +-1 / 0 on the bit pattern): the inputs are binary32, so this is the smallest change of the problem.
    The loss's gradient jumps at bilinear-cell borders and Adam normalises the step, so such last-bit differences are not
    damped but carried on.  Returns (farthest rotation, farthest translation, all draws).  No kernel-shaped code takes part:
    the oracle's binary32-position variant is not run here."""
    import oracle
    kw = dict(early_stop=0)
    kw.update(cfg_kw or {})
    runs = []
    rng = np.random.default_rng(seed)
    for _ in range(draws):
        bits = scene.poses_init.copy().view(np.int32) + rng.integers(-1, 2, size=scene.poses_init.shape).astype(np.int32)
        op = oracle.Optimizer(prob, bits.view(np.float32), scene.pairs, oracle_config(coord_fp32=0, **kw))
        op.run(iters)
        runs.append(pose_errors(op.poses, o64_poses))
    return max(r[0] for r in runs), max(r[1] for r in runs), runs


# Free-running rule (reading P7): the library's run may end no farther from the all-double oracle than the
# contract's 1e-3 degrees / 1e-4 scene units, or -- where correct runs of this very loop end farther apart than that -- than
# TWICE the farthest of the perturbed all-double runs above.  Why a factor at all: the draws and the library's run are
# samples of one heavy-tailed quantity (a chaotic divergence), and a ninth sample exceeds the largest of eight with
# probability 1/9 -- over the eight scenes of the suite a bare "no farther than the farthest" would fail a CORRECT
# implementation about once.  Why 2: the draws of one scene spread over a factor 3 to 10 (recorded in DESIGN.md P7).
SPREAD_FACTOR = 2.0


def within_spread(rot, tr, srot, str_):
    return rot <= max(1e-3, SPREAD_FACTOR * srot) and tr <= max(1e-4, SPREAD_FACTOR * str_)


def oracle_eval(prob, poses, pairs, lam, z_min=Z_MIN):
    """All-double oracle evaluation plus its event slack: (ref, slack)."""
    import oracle
    ref = oracle.loss_grad(prob, poses, pairs, lam, z_min=z_min, want_pair_G=True)
    return ref, oracle.event_slack(prob, poses, pairs, lam, ref, z_min=z_min)


def check_loss_grad(got, ref, sl, rtol_loss=1e-5, rtol_grad=1e-4, what=""):
    """The contract against the all-double oracle with the oracle's own event slack (module docstring).
    Returns a report: observed errors, slack sizes, and how many pairs / cameras needed any slack."""
    pv, pl, g = got["pair_valid"], got["pair_loss"].astype(np.float64), got["grad"].astype(np.float64)
    rv, rl, rg = ref["pair_valid"], ref["pair_loss"], ref["grad"]
    assert np.all(np.isfinite(sl["cam"])) and np.all(np.isfinite(sl["pair_loss"])), "unbounded slack (a depth at z_min)"
    assert np.all(pv >= rv - sl["k_out"]) and np.all(pv <= rv + sl["k_in"]), \
        (what, "valid counts differ beyond the samples the oracle flags at the validity border")
    err_l = np.abs(pl - rl)
    tol_l = rtol_loss * np.abs(rl) + sl["pair_loss"] + 1e-12
    w = int(np.argmax(err_l - tol_l))
    assert np.all(err_l <= tol_l), (what, "pair loss", w, pl[w], rl[w], err_l[w], tol_l[w])
    # reading T2: relative to the gradient's norm, or to the root-sum-square of its terms where they have cancelled
    # below it (near a minimum |g| -> 0 and "relative to |g|" would ask fp32 for more digits than its terms carry)
    err_g = np.linalg.norm(g - rg, axis=1); nrm = np.maximum(np.linalg.norm(rg, axis=1), sl["rss"])
    tol_g = rtol_grad * nrm + sl["cam"] + 1e-12
    c = int(np.argmax(err_g - tol_g))
    assert np.all(err_g <= tol_g), (what, "camera gradient", c, err_g[c] / nrm[c], sl["cam"][c] / nrm[c])
    assert abs(got["loss"] - ref["loss"]) <= rtol_loss * abs(ref["loss"]) + float(np.mean(sl["pair_loss"])) + 1e-12
    live = nrm > 0
    rep = dict(
        pair_loss_rel=float(np.max(err_l / np.maximum(np.abs(rl), 1e-30))),
        pairs_needing_slack=float(np.mean(err_l > rtol_loss * np.abs(rl) + 1e-12)),
        grad_rel=float(np.max(err_g[live] / nrm[live])) if live.any() else 0.0,
        grad_rel_median=float(np.median(err_g[live] / nrm[live])) if live.any() else 0.0,
        cams_needing_slack=float(np.mean(err_g > rtol_grad * nrm + 1e-12)),
        slack_rel_max=float(np.max(sl["cam"][live] / nrm[live])) if live.any() else 0.0,
        slack_rel_median=float(np.median(sl["cam"][live] / nrm[live])) if live.any() else 0.0,
        flagged_frac=float(sl["flagged"].sum() / max(int(rv.sum()), 1)))
    return rep


def assert_slack_is_small(rep, what=""):
    """Guards on the slack rule, set from what the B200 runs of round 3 show on all nine scenes (reading T1 has the
    table; observed maxima in brackets):
      - at most 0.2 % of the valid samples are flagged                        [0.14 %]
      - at most 0.5 % of the pairs need any slack for their loss              [0.2 %]
      - the median camera's slack is at most 5 % of its gradient scale        [3.3 %, orbit8 at lambda 6]
      - the median camera's ERROR is at most 1e-4 + a tenth of the median slack [ratio error : slack 0.006 .. 0.043]: the
        slack is a bound on what the flagged samples could move, and a correct kernel uses a small part of it -- a
        systematic gradient error of a few 1e-3 relative fails here even where every camera has flagged samples."""
    assert rep["flagged_frac"] <= 2e-3, (what, rep)
    assert rep["pairs_needing_slack"] <= 5e-3, (what, rep)
    assert rep["slack_rel_median"] <= 5e-2, (what, rep)
    assert rep["grad_rel_median"] <= 1e-4 + 0.1 * rep["slack_rel_median"], (what, rep)


def fmt_report(rep):
    return (f"pair loss rel err {rep['pair_loss_rel']:.1e} ({100 * rep['pairs_needing_slack']:.1f} % of pairs beyond 1e-5); camera grad rel err "
            f"max {rep['grad_rel']:.1e} median {rep['grad_rel_median']:.1e} ({100 * rep['cams_needing_slack']:.0f} % of cameras beyond 1e-4; "
            f"oracle slack max {rep['slack_rel_max']:.1e} median {rep['slack_rel_median']:.1e}); {100 * rep['flagged_frac']:.3f} % of samples flagged")


def pose_errors_per_camera(P_got, P_ref):
    """(rotation difference in degrees [N], translation difference in scene units [N])."""
    A = np.asarray(P_got, np.float64).reshape(-1, 3, 4); B = np.asarray(P_ref, np.float64).reshape(-1, 3, 4)
    rot = np.empty(len(A))
    for i, (a, b) in enumerate(zip(A, B)):
        R = a[:, :3] @ b[:, :3].T
        # angle from the skew part (well conditioned near zero)
        s = 0.5 * math.sqrt((R[2, 1] - R[1, 2]) ** 2 + (R[0, 2] - R[2, 0]) ** 2 + (R[1, 0] - R[0, 1]) ** 2)
        c = 0.5 * (np.trace(R) - 1.0)
        rot[i] = math.degrees(math.atan2(s, c))
    tr = np.linalg.norm(A[:, :, 3] - B[:, :, 3], axis=1)
    return rot, tr


def pose_errors(P_got, P_ref):
    """(max rotation difference in degrees, max translation difference in scene units)."""
    rot, tr = pose_errors_per_camera(P_got, P_ref)
    return float(rot.max()), float(tr.max())


class AdamBound:
    """What a bounded gradient error can do to an Adam increment (lock-step tests).

    Both sides run Adam on their own gradient history, evaluated at the same poses: the oracle on
    g_s, the library on g_s + e_s with |e_s| <= b_s per coordinate (b_s = 1e-4 |g_c| + the oracle's event slack of
    camera c).  Then, coordinate-wise,
        |m' - m| <= dm,  dm <- beta1 dm + (1 - beta1) b          |v' - v| <= dv,  dv <- beta2 dv + (1 - beta2)(2 |g| b + b^2)
        sqrt(v_hat') >= s_lo = sqrt(max(v_hat - dv_hat, 0)),      |sqrt(v_hat') - sqrt(v_hat)| <= s - s_lo   (concavity)
        |eps' - eps| <= lr [ dm_hat / (s_lo + eps_adam) + |m_hat| (s - s_lo) / ((s + eps_adam)(s_lo + eps_adam)) ]
    capped by |eps| + 8 lr (an Adam increment never exceeds ~7.3 lr sqrt(c2) / c1)."""

    def __init__(self, shape, beta1, beta2, adam_eps):
        self.b1, self.b2, self.eps = beta1, beta2, adam_eps
        self.dm = np.zeros(shape); self.dv = np.zeros(shape)

    def step(self, g, b, m, v, s, lr, inc):
        """g, b: this step's oracle gradient and error bound; m, v: the oracle's moments AFTER its update; s: 0-based
        step; inc: the oracle's increment.  Returns the bound on |increment_library - inc| per coordinate."""
        self.dm = self.b1 * self.dm + (1 - self.b1) * b
        self.dv = self.b2 * self.dv + (1 - self.b2) * (2 * np.abs(g) * b + b * b)
        c1 = 1 - self.b1 ** (s + 1); c2 = 1 - self.b2 ** (s + 1)
        mh, vh, dmh, dvh = m / c1, v / c2, self.dm / c1, self.dv / c2
        sq = np.sqrt(vh); s_lo = np.sqrt(np.maximum(vh - dvh, 0.0))
        de = lr * (dmh / (s_lo + self.eps) + np.abs(mh) * (sq - s_lo) / ((sq + self.eps) * (s_lo + self.eps)))
        return np.minimum(de, np.abs(inc) + 8 * lr)


def lockstep(sc, e, iters, ocfg, budget=0, seed=0, prob=None, label=""):
    """One-step-ahead parity against the ALL-DOUBLE oracle.  The loss has gradient jumps at bilinear-cell borders and
    Adam keeps stepping by ~lr once converged, so two free-running trajectories that differ by 1e-9 decorrelate after a
    few dozen iterations whatever the implementation.  Here the oracle is therefore re-started at every iteration from
    the library's own fp64 poses; its Adam moments are its own, fed with its own gradients.  At EVERY iteration:
      - the library's loss / valid counts / gradient at those poses (epo_loss_grad with lambda_k) against the oracle
        with the event slack (check_loss_grad);
      - the library's update (epo_step(1)) against the oracle's predicted poses: 1e-3 degrees and 1e-4 scene units plus
        what the gradient bound of this and the previous steps can move the Adam increment by (AdamBound);
      - theta95 (Eq. 9-10) and the loss trace; the phase, decided by the oracle's rule on the oracle's own theta / loss.
    Returns (worst, stop_at, iterations run)."""
    import oracle
    if prob is None:
        prob = oracle.preprocess(sc.K, sc.depth, sc.edges, z_min=Z_MIN)
    N = sc.n_views
    m = np.zeros((N, 6)); v = np.zeros((N, 6))
    ab = AdamBound((N, 6), ocfg.beta1, ocfg.beta2, ocfg.adam_eps)
    poses = e.get_poses_f64()
    worst = dict(rot=0.0, tr=0.0, rot_excess=0.0, tr_excess=0.0, theta=0.0, loss=0.0, grad=0.0, slack=0.0, allow_rot=0.0,
                 cells_beyond_contract=0, cells=0, ambiguous_phase=0)
    thetas = []; losses = []; phase = 0; stop_at = None; done = 1; k = -1
    for k in range(iters):
        lam, lr = oracle.lam_schedule(k, ocfg), oracle.lr_schedule(k, ocfg)
        # stochastic viewgraph sub-sampling: the oracle evaluates its own draw of step k
        pairs_k = sc.pairs[oracle.pair_subset(seed, k, len(sc.pairs), budget)] if budget else sc.pairs
        ref, sl = oracle_eval(prob, poses, pairs_k, lam)
        if not budget:                                   # epo_loss_grad always evaluates the full list
            rep = check_loss_grad(e.loss_grad(f32(lam)), ref, sl, what=f"{label} iteration {k}")
            worst["grad"] = max(worst["grad"], rep["grad_rel"]); worst["slack"] = max(worst["slack"], rep["slack_rel_max"])
        g = ref["grad"]
        b = np.repeat((1e-4 * np.maximum(np.linalg.norm(g, axis=1), sl["rss"]) + sl["cam"])[:, None], 6, axis=1)
        inc = oracle.adam(g.reshape(-1), m.reshape(-1), v.reshape(-1), k, lr, ocfg.beta1, ocfg.beta2, ocfg.adam_eps).reshape(N, 6)
        de = ab.step(g, b, m, v, k, lr, inc)
        pred = np.stack([oracle.se3_compose(oracle.se3_exp(inc[c]), poses[c]) for c in range(N)])
        th_pred = oracle.theta95(pred, poses)
        done, gphase = e.step(1)
        if done == 0:
            break
        new = e.get_poses_f64()
        loss, theta = e.get_trace(k, 1)
        rot, tr = pose_errors_per_camera(new, pred)
        t_norm = np.linalg.norm(pred.reshape(N, 3, 4)[:, :, 3], axis=1)
        a_rot = np.degrees(np.linalg.norm(de[:, 3:], axis=1))
        a_tr = np.linalg.norm(de[:, :3], axis=1) + np.linalg.norm(de[:, 3:], axis=1) * t_norm
        assert np.all(rot <= 1e-3 + 1.01 * a_rot) and np.all(tr <= 1e-4 + 1.01 * a_tr), \
            (label, k, float(rot.max()), float(a_rot.max()), float(tr.max()), float(a_tr.max()))
        worst["rot"] = max(worst["rot"], float(rot.max())); worst["tr"] = max(worst["tr"], float(tr.max()))
        worst["allow_rot"] = max(worst["allow_rot"], float(a_rot.max()))
        worst["cells_beyond_contract"] += int(np.sum((rot > 1e-3) | (tr > 1e-4))); worst["cells"] += N
        # theta95 = max of two 95th percentiles of per-camera angles: 1-Lipschitz in the largest per-camera change
        a_theta = float(max(a_rot.max(), np.degrees(np.max(a_tr / np.maximum(t_norm, 1e-12)))))
        th_err = abs(float(theta[0]) - th_pred)
        assert th_err <= 1e-3 * th_pred + 1e-7 + 1.01 * a_theta, (label, k, float(theta[0]), th_pred, a_theta)
        worst["theta"] = max(worst["theta"], th_err / max(th_pred, 1e-4 / 1e-3))
        l_tol = 1e-5 * abs(ref["loss"]) + float(np.mean(sl["pair_loss"])) + 1e-12
        assert abs(float(loss[0]) - ref["loss"]) <= l_tol, (label, k, float(loss[0]), ref["loss"])
        worst["loss"] = max(worst["loss"], abs(float(loss[0]) - ref["loss"]) / abs(ref["loss"]))
        # the stopping rule, run by the oracle on the oracle's own theta / loss values
        thetas.append(th_pred); losses.append(ref["loss"])
        want = phase
        if phase == 0:
            if oracle.converged(np.array(thetas), k, ocfg.w1, ocfg.eps1, ocfg.smooth_window): want = 1
        elif phase == 1 and (oracle.converged_loss(np.array(losses), k, ocfg.w_loss, ocfg.eps_loss) if ocfg.stop_rule == 1
                             else oracle.converged(np.array(thetas), k, ocfg.w2, ocfg.eps2, ocfg.smooth_window)):
            want = 2
        if gphase != want:
            # legitimate only if the library's own trace, run through the oracle's rule, gives the library's phase and
            # the two traces agree within the tolerance above (a threshold within rounding of theta95 / the loss)
            gl, gt = e.get_trace(0, k + 1)
            mine = phase
            if phase == 0:
                if oracle.converged(gt.astype(np.float64), k, ocfg.w1, ocfg.eps1, ocfg.smooth_window): mine = 1
            elif phase == 1 and (oracle.converged_loss(gl.astype(np.float64), k, ocfg.w_loss, ocfg.eps_loss) if ocfg.stop_rule == 1
                                 else oracle.converged(gt.astype(np.float64), k, ocfg.w2, ocfg.eps2, ocfg.smooth_window)):
                mine = 2
            assert mine == gphase, (label, k, gphase, want, mine)
            worst["ambiguous_phase"] += 1
            want = gphase
        phase = want
        if phase == 2 and stop_at is None:
            stop_at = k + 1
        poses = new
    return worst, stop_at, (k + 1 if done else k)


def fmt_lockstep(w):
    return (f"worst one-step differences: rot {w['rot']:.2e} deg, trans {w['tr']:.2e}, theta95 rel {w['theta']:.2e}, loss rel {w['loss']:.2e}; "
            f"gradient rel err max {w['grad']:.1e} (oracle slack up to {w['slack']:.1e}); {w['cells_beyond_contract']} of {w['cells']} "
            f"(iteration, camera) cells beyond the bare 1e-3 deg / 1e-4 (allowance up to {w['allow_rot']:.1e} deg); "
            f"{w['ambiguous_phase']} phase decisions within rounding of a threshold")
