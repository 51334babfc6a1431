#!/usr/bin/env python
"""Writes tests/golden/tiny_expected.txt: loss, per-pair losses / valid counts and per-camera gradients of
BASELINE.json config 1 (seeded Tiny scene) at its initial poses, for lambda = 10 and 6, and the poses after 200
fixed iterations -- as computed by the all-double CPU ORACLE, with the oracle's own event slack (reading T1:
what a binary32 evaluation may decide differently; for this scene a handful of samples).

Calls only `oracle/` and `epo_scenes/` (never the CUDA path).  Re-run after a justified change of the oracle:
    python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)


def main():
    import oracle
    from epo_scenes import make_scene
    f32 = lambda x: float(np.float32(x))
    sc = make_scene(1)
    zmin = f32(1e-6)
    prob = oracle.preprocess(sc.K, sc.depth, sc.edges, z_min=zmin)
    out = ["# written by tests/golden/make_golden.py from oracle/ only (config 1, all-double oracle + its event slack)"]
    out.append("edge_off " + " ".join(str(int(x)) for x in prob.edge_off))
    for lam in (10.0, 6.0):
        r = oracle.loss_grad(prob, sc.poses_init.astype(np.float64), sc.pairs, lam, z_min=zmin, want_pair_G=True)
        sl = oracle.event_slack(prob, sc.poses_init.astype(np.float64), sc.pairs, lam, r, z_min=zmin)
        out.append(f"lambda {lam!r}")
        out.append("loss " + repr(float(r["loss"])))
        out.append("pair_valid " + " ".join(str(int(x)) for x in r["pair_valid"]))
        out.append("pair_loss " + " ".join(repr(float(x)) for x in r["pair_loss"]))
        for c in range(sc.n_views):
            out.append(f"grad {c} " + " ".join(repr(float(x)) for x in r["grad"][c]))
        out.append("slack_k_out " + " ".join(str(int(x)) for x in sl["k_out"]))
        out.append("slack_k_in " + " ".join(str(int(x)) for x in sl["k_in"]))
        out.append("slack_pair_loss " + " ".join(repr(float(x)) for x in sl["pair_loss"]))
        out.append("slack_cam " + " ".join(repr(float(x)) for x in sl["cam"]))
    cfg = oracle.Config(lr_max=f32(3e-3), beta1=f32(0.9), beta2=f32(0.999), adam_eps=f32(1e-8), eps1=f32(0.5),
                        eps2=f32(0.1), z_min=zmin, early_stop=0)
    opt = oracle.Optimizer(prob, sc.poses_init, sc.pairs, cfg)
    assert opt.run(200)[0] == 200
    for c in range(sc.n_views):
        out.append(f"pose200 {c} " + " ".join(repr(float(x)) for x in np.asarray(opt.poses).reshape(-1, 12)[c]))
    out.append("loss_trace_0_199 " + repr(float(opt.loss[0])) + " " + repr(float(opt.loss[199])))
    with open(os.path.join(ROOT, "tests", "golden", "tiny_expected.txt"), "w") as f:
        f.write("\n".join(out) + "\n")


if __name__ == "__main__":
    main()
