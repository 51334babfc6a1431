"""GPU parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by element on the
same seeded inputs.  Run on the B200 box with `pytest -m gpu`."""
import numpy as np
import pytest

import oracle
from epo_scenes import SplitMix64, make_scene
from parity_utils import (Z_MIN, check_camera_grads, check_pair_losses, make_ctx, oracle_config, pose_errors)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _need_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2607_00579_b200 import build
    build.build()


SMALL = {  # reduced versions of BASELINE.json's configs: several tiles, ragged tails, seconds for the oracle
    "tiny": dict(config=1),
    "room6": dict(config=2, n_views=6),
    "orbit8": dict(config=3, n_views=8, overrides=dict(pairs=("knn", 4))),
    "room5_294": dict(config=4, n_views=5),
    "orbit10_dense": dict(config=5, n_views=10, overrides=dict(pairs=("knn", 5), early_stop=0)),
}
_scenes = {}


def scene(name):
    if name not in _scenes:
        _scenes[name] = make_scene(**SMALL[name])
    return _scenes[name]


# ------------------------------------------------------------------------------------ preprocessing
@pytest.mark.parametrize("name", list(SMALL))
def test_preprocessing_bit_exact(name):
    sc = scene(name)
    e = make_ctx(sc)
    prob = oracle.preprocess(sc.K, sc.depth, sc.edges, z_min=Z_MIN)
    off = e.get_edge_counts()
    assert np.array_equal(off, prob.edge_off)
    for i in range(sc.n_views):
        n = off[i + 1] - off[i]
        uv, z = e.get_edge_list(i, n)
        assert np.array_equal(uv, prob.uv[off[i]:off[i + 1]]) and np.array_equal(z, prob.z[off[i]:off[i + 1]])
        assert np.array_equal(e.get_dtf(i), prob.dtf[i]), (name, i)
    cp, perm = e.get_pair_order()
    ocp, operm = oracle.canonical_pairs(sc.pairs)
    assert np.array_equal(cp, ocp) and np.array_equal(perm, operm)
    e.destroy()


def test_preprocessing_adversarial_inputs():
    """Empty and full masks, single pixels, invalid depths, non-multiple-of-32 sizes, e_max sub-sampling."""
    from epo_scenes import Scene
    rng = SplitMix64(77)
    N, H, W = 7, 37, 45
    edges = np.zeros((N, H, W), np.uint8)
    edges[1] = 1                                                 # full
    edges[2, 17, 31] = 255                                       # one pixel
    edges[3] = (rng.uniform(H * W).reshape(H, W) < 0.02)
    edges[4] = (rng.uniform(H * W).reshape(H, W) < 0.5)
    edges[5, :, 0] = 1; edges[5, 0, :] = 1                       # border only
    edges[6, 5, :] = 1                                           # one full row: other rows use the sentinel
    depth = rng.uniform(N * H * W, 0.5, 4.0).reshape(N, H, W).astype(np.float32)
    depth[4, ::3, ::2] = np.nan; depth[4, 1::3, 1::2] = np.inf; depth[4, 2::3, ::5] = 0.0; depth[4, 5, 5] = -2.0
    depth[4, 6, 6] = 1e-7
    K = np.tile(np.array([40.0, 41.0, 22.0, 18.0], np.float32), (N, 1))
    poses = np.tile(np.eye(4, dtype=np.float32)[:3].reshape(12), (N, 1))
    pairs = np.array([[0, 1], [1, 0], [4, 3], [3, 4], [4, 3], [2, 6]], np.int32)
    sc = Scene("adv", W, H, K, poses.astype(np.float64), poses, depth, edges, pairs, {})
    for e_max in (0, 50):
        e = make_ctx(sc, e_max=e_max)
        prob = oracle.preprocess(K, depth, edges, z_min=Z_MIN, e_max=e_max)
        off = e.get_edge_counts()
        assert np.array_equal(off, prob.edge_off)
        assert off[1] - off[0] == 0                              # empty view: legal, DTF = W + H everywhere
        for i in range(N):
            uv, z = e.get_edge_list(i, off[i + 1] - off[i])
            assert np.array_equal(uv, prob.uv[off[i]:off[i + 1]]) and np.array_equal(z, prob.z[off[i]:off[i + 1]])
            assert np.array_equal(e.get_dtf(i), prob.dtf[i]), i
        assert np.all(e.get_dtf(0) == W + H)
        cp, perm = e.get_pair_order()
        ocp, operm = oracle.canonical_pairs(pairs)
        assert np.array_equal(cp, ocp) and np.array_equal(perm, operm)   # duplicates kept, stable
        got = e.loss_grad(10.0)                                           # pairs from an empty source give 0
        ref = oracle.loss_grad(prob, poses.astype(np.float64), pairs, 10.0, z_min=Z_MIN)
        assert got["pair_valid"][0] == 0 and got["pair_loss"][0] == 0.0
        check_pair_losses(got["pair_loss"], got["pair_valid"], ref, 10.0, max_event_frac=1.0)
        e.destroy()


def test_fp16_field_is_rne_of_fp32_field():
    sc = scene("room5_294")
    e = make_ctx(sc, dtf_format=1)
    ref = oracle.round_to_half(oracle.edt(sc.edges))
    for i in range(sc.n_views):
        assert np.array_equal(e.get_dtf(i), ref[i])
    e.destroy()


# ---------------------------------------------------------------------------------- loss + gradient
@pytest.mark.parametrize("name", list(SMALL))
@pytest.mark.parametrize("lam", [10.0, 6.0])
def test_loss_and_gradient_parity(name, lam):
    sc = scene(name)
    e = make_ctx(sc)
    prob = oracle.preprocess(sc.K, sc.depth, sc.edges, z_min=Z_MIN)
    got = e.loss_grad(lam)
    ref = oracle.loss_grad(prob, sc.poses_init.astype(np.float64), sc.pairs, lam, z_min=Z_MIN)
    worst = check_pair_losses(got["pair_loss"], got["pair_valid"], ref, lam)
    assert abs(got["loss"] - ref["loss"]) <= 1e-5 * abs(ref["loss"])
    gworst = check_camera_grads(got["grad"], ref["grad"])
    print(f"{name} lam={lam}: pair loss rel err {worst:.2e}, camera grad rel err {gworst:.2e}")
    # the evaluation must not move the state
    again = e.loss_grad(lam)
    assert abs(again["loss"] - got["loss"]) <= 1e-6 * abs(got["loss"])
    e.destroy()


def test_loss_and_gradient_parity_device_pointers():
    """Same call with CUDA tensors as inputs and outputs (no host synchronisation inside the call)."""
    import torch
    sc = scene("room6")
    e = make_ctx(sc, device_inputs=True)
    loss = torch.zeros(1, device="cuda"); pl = torch.zeros(e.P, device="cuda")
    pv = torch.zeros(e.P, dtype=torch.int32, device="cuda"); g = torch.zeros(sc.n_views, 6, device="cuda")
    e.loss_grad_into(8.0, loss, pl, pv, g)
    torch.cuda.synchronize()
    host = e.loss_grad(8.0)
    assert np.array_equal(pv.cpu().numpy(), host["pair_valid"])
    assert np.allclose(pl.cpu().numpy(), host["pair_loss"], rtol=1e-6, atol=0)
    assert np.allclose(g.cpu().numpy(), host["grad"], rtol=1e-5, atol=1e-9)
    prob = oracle.preprocess(sc.K, sc.depth, sc.edges, z_min=Z_MIN)
    ref = oracle.loss_grad(prob, sc.poses_init.astype(np.float64), sc.pairs, 8.0, z_min=Z_MIN)
    check_pair_losses(pl.cpu().numpy(), pv.cpu().numpy(), ref, 8.0)
    check_camera_grads(g.cpu().numpy(), ref["grad"])
    e.destroy()


def test_fp16_fields_against_fp32_oracle():
    """BASELINE.json config 4 variant: fp16 distance fields checked against the fp32 oracle at 1e-3 relative."""
    sc = scene("room5_294")
    e = make_ctx(sc, dtf_format=1)
    prob = oracle.preprocess(sc.K, sc.depth, sc.edges, z_min=Z_MIN)
    got = e.loss_grad(10.0)
    ref = oracle.loss_grad(prob, sc.poses_init.astype(np.float64), sc.pairs, 10.0, z_min=Z_MIN)
    check_pair_losses(got["pair_loss"], got["pair_valid"], ref, 10.0, rtol=1e-3)
    assert abs(got["loss"] - ref["loss"]) <= 1e-3 * abs(ref["loss"])
    # and exactly (1e-5) against the oracle run on the RNE-rounded field: the kernel samples that field
    prob_h = oracle.preprocess(sc.K, sc.depth, sc.edges, z_min=Z_MIN, half=True)
    ref_h = oracle.loss_grad(prob_h, sc.poses_init.astype(np.float64), sc.pairs, 10.0, z_min=Z_MIN)
    check_pair_losses(got["pair_loss"], got["pair_valid"], ref_h, 10.0)
    check_camera_grads(got["grad"], ref_h["grad"])
    e.destroy()


# ------------------------------------------------------------------------------------- optimisation
@pytest.mark.parametrize("name,iters", [("tiny", 200), ("room6", 200), ("orbit8", 60)])
def test_fixed_iteration_trajectory_parity(name, iters):
    """Final poses after a fixed number of iterations: 1e-3 degrees, 1e-4 scene units."""
    sc = scene(name)
    e = make_ctx(sc, early_stop=0)
    prob = oracle.preprocess(sc.K, sc.depth, sc.edges, z_min=Z_MIN)
    opt = oracle.Optimizer(prob, sc.poses_init, sc.pairs, oracle_config(early_stop=0))
    done, phase = e.step(iters)
    odone, _ = opt.run(iters)
    assert done == odone == iters
    rot, tr = pose_errors(e.get_poses_f64(), opt.poses)
    loss, theta = e.get_trace(0, iters)
    lrel = np.max(np.abs(loss - opt.loss[:iters]) / np.abs(opt.loss[:iters]))
    trel = np.max(np.abs(theta - opt.theta[:iters]) / np.maximum(np.abs(opt.theta[:iters]), 1e-4))
    print(f"{name}: after {iters} its rot diff {rot:.2e} deg, trans diff {tr:.2e}, loss trace rel {lrel:.2e}, theta rel {trel:.2e}")
    assert rot <= 1e-3 and tr <= 1e-4
    assert lrel <= 1e-4
    assert np.allclose(e.get_poses(), e.get_poses_f64().astype(np.float32))
    e.destroy()


def test_early_stop_parity():
    """Config-5-like run with the stopping rule active: theta95 traces agree up to the earlier stop, the
    stop steps differ by at most 2, phase 2 is reported, and epo_step does nothing once stopped."""
    sc = scene("orbit10_dense")
    kw = dict(w1=10, w2=20, eps1=0.5, eps2=0.12, early_stop=1)      # shortened windows: same rule, test-sized run
    e = make_ctx(sc, **kw)
    prob = oracle.preprocess(sc.K, sc.depth, sc.edges, z_min=Z_MIN)
    opt = oracle.Optimizer(prob, sc.poses_init, sc.pairs, oracle_config(**{k: (float(np.float32(v)) if isinstance(v, float) else v) for k, v in kw.items()}))
    done, phase = e.step(600)
    odone, _ = opt.run(600)
    assert phase == 2 and opt.phase.value == 2 and done < 600
    assert abs(done - odone) <= 2, (done, odone)
    k = min(done, odone)
    _, theta = e.get_trace(0, k)
    assert np.all(np.abs(theta - opt.theta[:k]) <= np.maximum(1e-3 * np.abs(opt.theta[:k]), 1e-4))
    assert e.step(5) == (0, 2)
    e.reset()                                                           # back to the initial poses, state cleared
    done2, _ = e.step(done)
    assert done2 == done
    e.destroy()


def test_step_in_pieces_equals_one_call():
    sc = scene("tiny")
    a = make_ctx(sc, early_stop=0); b = make_ctx(sc, early_stop=0)
    a.step(30)
    for n in (1, 9, 20):
        b.step(n, sync=False)
    rot, tr = pose_errors(a.get_poses_f64(), b.get_poses_f64())
    assert rot < 1e-9 and tr < 1e-12
    a.destroy(); b.destroy()


# ------------------------------------------------------------------------------------------- errors
def test_error_codes():
    import ctypes as C
    import paper_2607_00579_b200 as pkg
    sc = scene("tiny")
    cfg = pkg.epo_config_default(n_views=sc.n_views, width=sc.W, height=sc.H)
    e = pkg.Epo(cfg)
    L = pkg.lib()
    assert L.epo_set_pairs(e._h, sc.pairs.ctypes.data, len(sc.pairs)) == pkg.EPO_ERR_BAD_STATE
    out = np.zeros(1, np.float32)
    assert L.epo_loss_grad(e._h, C.c_float(10.0), out.ctypes.data, None, None, None) == pkg.EPO_ERR_BAD_STATE
    assert L.epo_step(e._h, 1, None, None) == pkg.EPO_ERR_BAD_STATE
    assert L.epo_set_views(e._h, None, None, None, None) == pkg.EPO_ERR_INVALID_ARG
    badK = sc.K.copy(); badK[1, 0] = -1.0
    assert L.epo_set_views(e._h, badK.ctypes.data, sc.poses_init.ctypes.data, sc.depth.ctypes.data, sc.edges.ctypes.data) == pkg.EPO_ERR_INVALID_ARG
    assert b"intrinsics" in L.epo_last_error(e._h)
    e.set_views(sc.K, sc.poses_init, sc.depth, sc.edges)
    assert L.epo_loss_grad(e._h, C.c_float(10.0), out.ctypes.data, None, None, None) == pkg.EPO_ERR_BAD_STATE
    for bad in ([[0, 0]], [[0, 4]], [[-1, 2]]):
        bp = np.array(bad, np.int32)
        assert L.epo_set_pairs(e._h, bp.ctypes.data, 1) == pkg.EPO_ERR_INVALID_ARG
    assert L.epo_set_pairs(e._h, sc.pairs.ctypes.data, 0) == pkg.EPO_ERR_INVALID_ARG
    e.set_pairs(sc.pairs)
    good = e.loss_grad(10.0)["loss"]
    # a failed set_pairs leaves the context unchanged
    assert L.epo_set_pairs(e._h, np.array([[0, 0]], np.int32).ctypes.data, 1) == pkg.EPO_ERR_INVALID_ARG
    assert e.loss_grad(10.0)["loss"] == good
    assert L.epo_loss_grad(e._h, C.c_float(10.0), None, None, None, None) == pkg.EPO_ERR_INVALID_ARG
    assert L.epo_step(e._h, -1, None, None) == pkg.EPO_ERR_INVALID_ARG
    e.destroy()
