"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (same library build, same
work decomposition, device-resident inputs): every pair and every camera of configs 2-5 against the CPU oracle
(it is C + OpenMP, so whole evaluations at full size take seconds), plus bit-exact preprocessing on sampled
views and a few lock-step optimiser iterations."""
import numpy as np
import pytest

import oracle
from epo_scenes import make_scene
from parity_utils import Z_MIN, check_camera_grads, check_pair_losses, make_ctx, oracle_config, pose_errors

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _need_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2607_00579_b200 import build
    build.build()


def _full(config, **cfg_over):
    sc = make_scene(config)
    e = make_ctx(sc, device_inputs=True, **cfg_over)
    prob = oracle.preprocess(sc.K, sc.depth, sc.edges, z_min=Z_MIN)
    return sc, e, prob


@pytest.mark.parametrize("config", [2, 3, 4, 5])
def test_full_size_loss_gradient_and_preprocessing(config):
    sc, e, prob = _full(config, early_stop=0)
    N = sc.n_views
    # preprocessing: offsets of all views; lists and fields bit-exact on a seeded sample of views (+ first, last)
    off = e.get_edge_counts()
    assert np.array_equal(off, prob.edge_off)
    views = sorted({0, N - 1} | {int(v) for v in np.random.default_rng(config).choice(N, size=min(6, N), replace=False)})
    for i in views:
        uv, z = e.get_edge_list(i, off[i + 1] - off[i])
        assert np.array_equal(uv, prob.uv[off[i]:off[i + 1]]) and np.array_equal(z, prob.z[off[i]:off[i + 1]])
        assert np.array_equal(e.get_dtf(i), prob.dtf[i]), i
    cp, perm = e.get_pair_order()
    ocp, operm = oracle.canonical_pairs(sc.pairs)
    assert np.array_equal(cp, ocp) and np.array_equal(perm, operm)
    # loss + gradient, all pairs, all cameras
    poses = sc.poses_init.astype(np.float64)
    for lam in (10.0, 6.0):
        got = e.loss_grad(lam)
        ref32 = oracle.loss_grad(prob, poses, sc.pairs, lam, z_min=Z_MIN, coord_fp32=1)
        assert np.array_equal(got["pair_valid"], ref32["pair_valid"])
        w32 = check_pair_losses(got["pair_loss"], got["pair_valid"], ref32, lam, max_event_frac=0.0)
        assert abs(got["loss"] - ref32["loss"]) <= 1e-5 * abs(ref32["loss"])
        g32 = check_camera_grads(got["grad"], ref32["grad"])
        print(f"config {config} full size lam={lam}: {len(sc.pairs)} pairs, {int(got['pair_valid'].sum())} valid samples; "
              f"pair loss rel err {w32:.2e}, camera grad rel err {g32:.2e}")
    ref64 = oracle.loss_grad(prob, poses, sc.pairs, 10.0, z_min=Z_MIN)
    got = e.loss_grad(10.0)
    check_pair_losses(got["pair_loss"], got["pair_valid"], ref64, 10.0)
    # three lock-step iterations of the loop at full size
    ocfg = oracle_config(coord_fp32=1, early_stop=0)
    m = np.zeros((N, 6)); v = np.zeros((N, 6))
    P = e.get_poses_f64()
    for k in range(3):
        ref = oracle.loss_grad(prob, P, sc.pairs, oracle.lam_schedule(k, ocfg), z_min=Z_MIN, coord_fp32=1)
        inc = oracle.adam(ref["grad"].reshape(-1), m.reshape(-1), v.reshape(-1), k, oracle.lr_schedule(k, ocfg),
                          ocfg.beta1, ocfg.beta2, ocfg.adam_eps).reshape(N, 6)
        pred = np.stack([oracle.se3_compose(oracle.se3_exp(inc[c]), P[c]) for c in range(N)])
        assert e.step(1)[0] == 1
        new = e.get_poses_f64()
        rot, tr = pose_errors(new, pred)
        loss, theta = e.get_trace(k, 1)
        assert rot <= 1e-3 and tr <= 1e-4, (k, rot, tr)
        assert abs(float(loss[0]) - ref["loss"]) <= 1e-5 * abs(ref["loss"])
        th = oracle.theta95(pred, P)
        assert abs(float(theta[0]) - th) <= 1e-3 * th + 1e-7
        P = new
    e.destroy()


def test_full_size_config4_fp16_fields():
    """BASELINE.json config 4 variant: fp16 distance fields against the fp32 oracle at 1e-3 relative."""
    sc, e, prob = _full(4, dtf_format=1)
    poses = sc.poses_init.astype(np.float64)
    got = e.loss_grad(10.0)
    ref = oracle.loss_grad(prob, poses, sc.pairs, 10.0, z_min=Z_MIN)
    check_pair_losses(got["pair_loss"], got["pair_valid"], ref, 10.0, rtol=1e-3)
    assert abs(got["loss"] - ref["loss"]) <= 1e-3 * abs(ref["loss"])
    err = np.linalg.norm(got["grad"] - ref["grad"], axis=1) / np.linalg.norm(ref["grad"], axis=1)
    print(f"config 4 fp16 fields: loss rel err {abs(got['loss'] - ref['loss']) / ref['loss']:.2e}, camera grad rel err max {err.max():.2e}")
    # the fp16 field's gradient differs from the fp32 field's by the rounding of neighbouring taps (2^-11 relative
    # on values up to ~100 px against differences of ~1 px): reported, bounded loosely
    assert err.max() <= 5e-2
    e.destroy()


def test_full_size_config5_early_stop_runs_to_its_own_stop():
    """Config 5 as stated: early stop active, max 2000 steps, one epo_step call with no host sync inside."""
    sc, e, prob = _full(5, early_stop=1)
    done, phase = e.step(2000)
    loss, theta = e.get_trace(0, done)
    print(f"config 5 full size: stopped after {done} iterations in phase {phase}; loss {loss[0]:.4f} -> {loss[-1]:.4f}; "
          f"theta95 {theta[0]:.3f} -> {theta[-1]:.4f} deg")
    assert phase == 2 and 100 <= done < 2000
    assert loss[-1] < 0.5 * loss[0]
    # the rule, re-run by the oracle on the GPU's own theta trace, fires at exactly that step and not before
    ocfg = oracle_config(early_stop=1)
    th = theta.astype(np.float64); ph = 0; fired = None
    for s in range(done):
        if ph == 0:
            if oracle.converged(th, s, ocfg.w1, ocfg.eps1, ocfg.smooth_window): ph = 1
        elif ph == 1 and oracle.converged(th, s, ocfg.w2, ocfg.eps2, ocfg.smooth_window):
            ph = 2; fired = s + 1; break
    assert fired == done, (fired, done)
    assert e.step(10) == (0, 2)
    e.destroy()


def test_full_size_config4_stochastic_pair_subsampling():
    """Config 4's 39,800 pairs with the paper's budget M = 1024: the device draw equals the oracle's
    bit for bit, and three iterations on the drawn subsets match the oracle in lock-step."""
    M, seed = 1024, 2607
    sc, e, prob = _full(4, early_stop=0, pair_budget=M, subsample_seed=seed)
    Pn = len(sc.pairs)
    for step in (0, 1, 500):
        got = e.get_pair_subset(step)
        assert got.sum() == M and np.array_equal(got, oracle.pair_subset(seed, step, Pn, M)), step
    ocfg = oracle_config(coord_fp32=1, early_stop=0)
    N = sc.n_views
    m = np.zeros((N, 6)); v = np.zeros((N, 6))
    P = e.get_poses_f64()
    for k in range(3):
        pairs_k = sc.pairs[oracle.pair_subset(seed, k, Pn, M)]
        ref = oracle.loss_grad(prob, P, pairs_k, oracle.lam_schedule(k, ocfg), z_min=Z_MIN, coord_fp32=1)
        inc = oracle.adam(ref["grad"].reshape(-1), m.reshape(-1), v.reshape(-1), k, oracle.lr_schedule(k, ocfg),
                          ocfg.beta1, ocfg.beta2, ocfg.adam_eps).reshape(N, 6)
        pred = np.stack([oracle.se3_compose(oracle.se3_exp(inc[c]), P[c]) for c in range(N)])
        assert e.step(1)[0] == 1
        new = e.get_poses_f64()
        rot, tr = pose_errors(new, pred)
        loss, _ = e.get_trace(k, 1)
        assert rot <= 1e-3 and tr <= 1e-4, (k, rot, tr)
        assert abs(float(loss[0]) - ref["loss"]) <= 1e-5 * abs(ref["loss"]), (k, float(loss[0]), ref["loss"])
        P = new
    e.destroy()


def test_full_size_config3_viewgraph():
    """Config 3's 100 views: all 9,900 ordered cycles (31.5 M grid points at stride 8) bit-exact against the oracle."""
    import time
    sc, e, prob = _full(3)
    e.build_viewgraph()                                            # warm-up (allocations)
    t0 = time.perf_counter(); pairs, counts = e.build_viewgraph(stride=8, tau=3.0, min_frac=0.125, want_counts=True)
    t_gpu = time.perf_counter() - t0
    t0 = time.perf_counter()
    ref = oracle.viewgraph_counts(sc.K, sc.poses_init.astype(np.float64), sc.depth, stride=8, tau=3.0, z_min=Z_MIN, coord_fp32=1)
    t_cpu = time.perf_counter() - t0
    assert np.array_equal(counts, ref)
    assert np.array_equal(pairs, oracle.viewgraph_pairs(ref, 0.125))
    print(f"config 3 viewgraph: {len(pairs)} directed pairs of 9900; library call {1e3 * t_gpu:.2f} ms (incl. D2H of pairs "
          f"and counts), oracle {t_cpu:.2f} s on {oracle.num_threads()} threads")
    e.destroy()


def test_full_size_edge_extraction_config3_shape():
    """100 images at 518x392 (config 3's shape): Canny byte-exact against the oracle, with the wall time of both."""
    import time
    import torch
    from test_gpu_parity import _test_images
    from paper_2607_00579_b200 import Epo, epo_config_default
    base = _test_images(4, 392, 518, seed=3)
    imgs = np.ascontiguousarray(np.concatenate([np.roll(base, 7 * k, axis=2) for k in range(25)]))     # 100 images
    e = Epo(epo_config_default(n_views=100, width=518, height=392, stream=torch.cuda.current_stream().cuda_stream))
    d_img = torch.from_numpy(imgs).cuda(); d_out = torch.zeros_like(d_img)
    e.extract_edges(d_img, 12, 48, out=d_out); torch.cuda.synchronize()
    t0 = time.perf_counter(); e.extract_edges(d_img, 12, 48, out=d_out); torch.cuda.synchronize(); t_gpu = time.perf_counter() - t0
    t0 = time.perf_counter(); ref = oracle.canny(imgs, 12, 48); t_cpu = time.perf_counter() - t0
    assert np.array_equal(d_out.cpu().numpy(), ref)
    print(f"Canny, 100 x 518x392: library {1e3 * t_gpu:.2f} ms (device-resident), oracle {t_cpu:.2f} s on {oracle.num_threads()} "
          f"threads; {100 * ref.mean():.1f} % edge pixels")
    e.destroy()


def test_full_size_config3_joint_phase_gradients():
    """Config 3 at full size: d L / d ln f of all 100 cameras and d L / d Z of all 1.6 M edge pixels against the oracle."""
    import time
    sc, e, prob = _full(3)
    e.loss_grad_joint(10.0)
    t0 = time.perf_counter(); got = e.loss_grad_joint(10.0); t_gpu = time.perf_counter() - t0
    t0 = time.perf_counter()
    gf, gz = oracle.joint_grad(prob, sc.poses_init.astype(np.float64), sc.pairs, 10.0, z_min=Z_MIN, coord_fp32=1)
    t_cpu = time.perf_counter() - t0
    assert np.all(np.abs(got["g_logf"] - gf) <= 1e-4 * np.abs(gf) + 1e-9)
    worst = 0.0
    for i in range(sc.n_views):
        lo, hi = prob.edge_off[i], prob.edge_off[i + 1]
        u, v = prob.uv[lo:hi, 0].astype(int), prob.uv[lo:hi, 1].astype(int)
        mine, ref = got["g_depth"][i, v, u].astype(np.float64), gz[lo:hi]
        worst = max(worst, np.linalg.norm(mine - ref) / np.linalg.norm(ref))
    assert worst <= 1e-4
    print(f"config 3 joint gradients: d/dZ per-view rel err max {worst:.2e}; library call {1e3 * t_gpu:.1f} ms (incl. the D2H of "
          f"the 81 MB map), oracle {t_cpu:.1f} s (serial over pairs)")
    e.destroy()
