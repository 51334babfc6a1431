"""tests/golden fixtures: the paper's printed constants (cited), the closed-form schedule values that follow
from them, and oracle-written expected values of BASELINE.json config 1 (tests/golden/make_golden.py, which
calls only oracle/)."""
import math
import os

import numpy as np
import pytest

import oracle

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _rows(name):
    for ln in open(os.path.join(GOLD, name)):
        ln = ln.strip()
        if ln and not ln.startswith("#"):
            yield ln.split()


def load_tiny_expected():
    out = {"by_lambda": {}, "pose200": {}}
    cur = None
    for r in _rows("tiny_expected.txt"):
        k = r[0]
        if k == "edge_off":
            out["edge_off"] = np.array(r[1:], np.int32)
        elif k == "lambda":
            cur = out["by_lambda"].setdefault(float(r[1]), {"grad": {}})
        elif k == "loss":
            cur["loss"] = float(r[1])
        elif k == "pair_valid":
            cur["pair_valid"] = np.array(r[1:], np.int32)
        elif k == "pair_loss":
            cur["pair_loss"] = np.array(r[1:], np.float64)
        elif k == "grad":
            cur["grad"][int(r[1])] = np.array(r[2:], np.float64)
        elif k in ("slack_k_out", "slack_k_in"):
            cur[k] = np.array(r[1:], np.int32)
        elif k in ("slack_pair_loss", "slack_cam"):
            cur[k] = np.array(r[1:], np.float64)
        elif k == "pose200":
            out["pose200"][int(r[1])] = np.array(r[2:], np.float64)
        elif k == "loss_trace_0_199":
            out["loss_trace"] = (float(r[1]), float(r[2]))
    return out


def test_paper_constants_are_the_defaults_of_oracle_and_library():
    """PAPER.md:121, 123, 462 -> oracle.Config defaults and epo_config_default (no GPU needed for either)."""
    import paper_2607_00579_b200 as pkg
    vals = {r[0]: float(r[1]) for r in _rows("paper_constants.txt")}
    assert len(vals) == 12
    ocfg, lcfg = oracle.Config(), pkg.epo_config_default()
    for name, v in vals.items():
        assert abs(float(getattr(ocfg, name)) - v) <= 1e-15 * max(1.0, abs(v)), name
        assert abs(float(getattr(lcfg, name)) - v) <= 1e-7 * max(1.0, abs(v)), name       # fp32 fields


def test_schedules_hit_the_hand_computed_values():
    cfg = oracle.Config()
    n = 0
    for kind, s, v in _rows("schedules.txt"):
        got = oracle.lam_schedule(int(s), cfg) if kind == "lambda" else oracle.lr_schedule(int(s), cfg)
        assert abs(got - float(v)) <= 1e-12, (kind, s, got, v)
        n += 1
    assert n == 11
    # cosine branch end points (closed form): lr_s = lr_max/2 (1 + cos(pi (s-25)/1975))
    assert abs(oracle.lr_schedule(25 + 1975 // 5 * 0 + 0, cfg) - 3e-3) < 1e-18
    s = 1012                                                     # (s - 25)/1975 ~ 0.49975 -> just above lr_max/2
    assert abs(oracle.lr_schedule(s, cfg) - 1.5e-3 * (1 + math.cos(math.pi * 987 / 1975))) < 1e-15


def test_oracle_reproduces_its_stored_values(tiny_scene, tiny_problem):
    """Guards the oracle against silent drift: a change of its arithmetic must come with a regenerated fixture
    and a commit message that names the passage or DESIGN.md reading behind it."""
    exp = load_tiny_expected()
    sc = tiny_scene
    zmin = float(np.float32(1e-6))
    prob = oracle.preprocess(sc.K, sc.depth, sc.edges, z_min=zmin)
    assert np.array_equal(prob.edge_off, exp["edge_off"])
    for lam, e in exp["by_lambda"].items():
        r = oracle.loss_grad(prob, sc.poses_init.astype(np.float64), sc.pairs, lam, z_min=zmin, want_pair_G=True)
        sl = oracle.event_slack(prob, sc.poses_init.astype(np.float64), sc.pairs, lam, r, z_min=zmin)
        assert np.array_equal(sl["k_out"], e["slack_k_out"]) and np.array_equal(sl["k_in"], e["slack_k_in"])
        assert np.allclose(sl["cam"], e["slack_cam"], rtol=1e-11, atol=1e-15)
        assert np.allclose(sl["pair_loss"], e["slack_pair_loss"], rtol=1e-11, atol=1e-15)
        assert np.array_equal(r["pair_valid"], e["pair_valid"])
        assert np.allclose(r["pair_loss"], e["pair_loss"], rtol=1e-13, atol=0)
        assert abs(r["loss"] - e["loss"]) <= 1e-13 * abs(e["loss"])
        for c, g in e["grad"].items():
            assert np.allclose(r["grad"][c], g, rtol=1e-11, atol=1e-13)


@pytest.mark.gpu
def test_cuda_path_matches_the_stored_oracle_values(tiny_scene):
    """The CUDA path against values stored by the oracle-only script (nothing here is computed by the oracle at
    test time): per-pair loss 1e-5, per-camera gradient 1e-4 against the all-double oracle, plus only the stored
    event slack of the oracle's own flagged samples (reading T1); poses after 200 free-running iterations."""
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from parity_utils import make_ctx, pose_errors
    exp = load_tiny_expected()
    e = make_ctx(tiny_scene, early_stop=0)
    assert np.array_equal(e.get_edge_counts(), exp["edge_off"])
    for lam, ref in exp["by_lambda"].items():
        got = e.loss_grad(lam)
        assert np.all(got["pair_valid"] >= ref["pair_valid"] - ref["slack_k_out"])
        assert np.all(got["pair_valid"] <= ref["pair_valid"] + ref["slack_k_in"])
        assert np.all(np.abs(got["pair_loss"] - ref["pair_loss"]) <= 1e-5 * np.abs(ref["pair_loss"]) + ref["slack_pair_loss"])
        assert abs(got["loss"] - ref["loss"]) <= 1e-5 * abs(ref["loss"]) + ref["slack_pair_loss"].mean()
        for c, g in ref["grad"].items():
            assert np.linalg.norm(got["grad"][c] - g) <= 1e-4 * np.linalg.norm(g) + ref["slack_cam"][c]
    assert e.step(200)[0] == 200
    P = np.stack([exp["pose200"][c] for c in range(tiny_scene.n_views)])
    rot, tr = pose_errors(e.get_poses_f64(), P)
    assert rot <= 1e-3 and tr <= 1e-4, (rot, tr)
    loss, _ = e.get_trace(0, 200)
    assert abs(loss[0] - exp["loss_trace"][0]) <= 1e-5 * exp["loss_trace"][0]
    e.destroy()
