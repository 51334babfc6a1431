"""Shared helpers of the GPU parity tests: build a library context from a Scene, and compare its
outputs with the CPU oracle under BASELINE.json's tolerances.

Tolerances (BASELINE.json north_star): edge lists / pair lists / EDT bit-exact; per-pair loss 1e-5
relative; per-camera gradient 1e-4 relative; poses after a fixed 200 iterations 1e-3 degrees and
1e-4 scene units.  "Tolerance realism": a sample the fp64 oracle places within 1e-3 px of
the validity border may be decided the other way by the fp32 kernel; such a flip moves a pair loss by
at most rho(lambda)/n_valid, so pairs where the oracle reports k such samples get that much slack,
and the tests assert that these pairs are a small minority.
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


def huber(d, delta=1.0):
    return 0.5 * d * d if d <= delta else delta * (d - 0.5 * delta)


def check_pair_losses(got_loss, got_valid, ref, lam, rtol=1e-5, delta=1.0, max_event_frac=0.2):
    """Per-pair loss 1e-5 relative; pairs with oracle-flagged border samples get k rho(lambda)/n slack."""
    ref_loss, ref_valid, near = ref["pair_loss"], ref["pair_valid"], ref["near"]
    rho_max = huber(min(lam, 1e30), delta)
    nb = near[:, 0]
    assert np.all(np.abs(got_valid - ref_valid) <= nb), "valid counts differ beyond flagged border samples"
    tol = rtol * np.abs(ref_loss) + nb * rho_max / np.maximum(ref_valid, 1) + 1e-12
    err = np.abs(got_loss.astype(np.float64) - ref_loss)
    worst = int(np.argmax(err / tol))
    assert np.all(err <= tol), (worst, got_loss[worst], ref_loss[worst], err[worst], tol[worst], nb[worst])
    clean = nb == 0
    assert clean.mean() >= 1 - max_event_frac, "too many pairs needed the border-event slack"
    rel = err[clean] / np.maximum(np.abs(ref_loss[clean]), 1e-30)
    return float(rel.max()) if clean.any() else 0.0


def check_camera_grads(got_grad, ref_grad, rtol=1e-4):
    """Per-camera gradient: || g_gpu - g_oracle || <= 1e-4 || g_oracle || for every camera."""
    err = np.linalg.norm(got_grad.astype(np.float64) - ref_grad, axis=1)
    nrm = np.linalg.norm(ref_grad, axis=1)
    rel = err / np.maximum(nrm, 1e-30)
    assert np.all(err <= rtol * nrm + 1e-12), (int(np.argmax(rel)), rel.max())
    return float(rel.max())


def pose_errors(P_got, P_ref):
    """(max rotation difference in degrees, max translation difference in scene units)."""
    A = np.asarray(P_got, np.float64).reshape(-1, 3, 4); B = np.asarray(P_ref, np.float64).reshape(-1, 3, 4)
    rot = []
    for a, b in zip(A, B):
        R = a[:, :3] @ b[:, :3].T
        # angle from the skew part (well conditioned near zero)
        s = 0.5 * math.sqrt((R[2, 1] - R[1, 2]) ** 2 + (R[0, 2] - R[2, 0]) ** 2 + (R[1, 0] - R[0, 1]) ** 2)
        c = 0.5 * (np.trace(R) - 1.0)
        rot.append(math.degrees(math.atan2(s, c)))
    tr = np.linalg.norm(A[:, :, 3] - B[:, :, 3], axis=1)
    return float(np.max(rot)), float(np.max(tr))
