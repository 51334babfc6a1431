"""Pins for the oracle's preprocessing (O1, O2, O3; checks Z3).

Every expected value here comes from something OTHER than the oracle: the definition evaluated by
brute force in numpy, closed forms, scipy / numpy library routines.
"""
import itertools

import numpy as np
import pytest
import scipy.ndimage

import oracle
from epo_scenes import SplitMix64


def _numpy_bruteforce_edt(mask):
    """PAPER.md:62 'each pixel encodes the Euclidean distance to the nearest edge', by exhaustive search."""
    H, W = mask.shape
    ys, xs = np.nonzero(mask)
    if len(ys) == 0:
        return np.full((H, W), float(W + H), np.float32)
    yy, xx = np.mgrid[0:H, 0:W]
    d2 = (yy[..., None] - ys) ** 2 + (xx[..., None] - xs) ** 2
    return np.sqrt(d2.min(axis=2).astype(np.float64)).astype(np.float32)


def test_edt_all_3x3_masks_bit_exact():
    for bits in itertools.product([0, 1], repeat=9):
        m = np.array(bits, np.uint8).reshape(3, 3)
        ref = _numpy_bruteforce_edt(m)
        assert np.array_equal(oracle.edt_brute(m), ref)
        assert np.array_equal(oracle.edt(m), ref)


def test_edt_random_masks_vs_bruteforce_and_scipy():
    rng = SplitMix64(1234)
    for k in range(500):
        H = 2 + int(rng.integers(1, 23)[0]); W = 2 + int(rng.integers(1, 23)[0])
        mode = k % 4
        if mode == 0:      # a single edge pixel
            m = np.zeros((H, W), np.uint8); m[int(rng.integers(1, H)[0]), int(rng.integers(1, W)[0])] = 1
        elif mode == 1:    # ~2 %
            m = (rng.uniform(H * W).reshape(H, W) < 0.02).astype(np.uint8)
        elif mode == 2:    # 50 %
            m = (rng.uniform(H * W).reshape(H, W) < 0.5).astype(np.uint8)
        else:              # full
            m = np.ones((H, W), np.uint8)
        ref = _numpy_bruteforce_edt(m)
        got = oracle.edt(m)
        assert np.array_equal(got, ref), (k, H, W)
        assert np.array_equal(oracle.edt_brute(m), ref)
        if m.any():        # library cross-check (float64 -> cast)
            sp = scipy.ndimage.distance_transform_edt(m == 0).astype(np.float32)
            assert np.array_equal(got, sp)


def test_edt_closed_forms():
    H, W = 37, 53
    m = np.zeros((H, W), np.uint8); m[11, 29] = 1
    yy, xx = np.mgrid[0:H, 0:W]
    assert np.array_equal(oracle.edt(m), np.sqrt(((yy - 11) ** 2 + (xx - 29) ** 2).astype(np.float64)).astype(np.float32))
    m = np.zeros((H, W), np.uint8); m[:, 17] = 1           # full column c -> |x - c|
    assert np.array_equal(oracle.edt(m), np.abs(xx - 17).astype(np.float32))
    m = np.zeros((H, W), np.uint8)                          # empty -> W + H everywhere (reading S8)
    assert np.array_equal(oracle.edt(m), np.full((H, W), W + H, np.float32))
    m = np.zeros((H, W), np.uint8); m[5, :] = 1             # full row -> |y - 5|, rows without edges use sentinel
    assert np.array_equal(oracle.edt(m), np.abs(yy - 5).astype(np.float32))


def test_edt_full_resolution_against_scipy():
    """One 518x392 view (the 3DFM working resolution) against scipy's exact EDT."""
    rng = SplitMix64(99)
    m = (rng.uniform(392 * 518).reshape(392, 518) < 0.002).astype(np.uint8)
    m[200:260, 100:180] = 0
    sp = scipy.ndimage.distance_transform_edt(m == 0).astype(np.float32)
    assert np.array_equal(oracle.edt(m), sp)
    batch = np.stack([m, np.zeros_like(m), m[::-1].copy()])
    got = oracle.edt(batch)
    assert np.array_equal(got[0], sp) and np.all(got[1] == 518 + 392)
    assert np.array_equal(got[2], sp[::-1])


def test_round_to_half_matches_numpy_float16():
    rng = SplitMix64(5)
    x = np.concatenate([rng.uniform(20000, 0, 700).astype(np.float32),
                        np.sqrt(np.arange(0, 70000, dtype=np.float64)).astype(np.float32),
                        np.array([0.0, 1e-8, 6e-8, 3e-5, 6.1e-5, 65504.0, 65519.9, 65520.0, 1e6, 2049.0, 2051.0],
                                 np.float32)])
    with np.errstate(over="ignore"):
        ref = x.astype(np.float16).astype(np.float32)
    assert np.array_equal(oracle.round_to_half(x), ref)


def test_edge_list_raster_order_and_depth_filter():
    rng = SplitMix64(7)
    H, W = 19, 23
    edges = (rng.uniform(H * W).reshape(H, W) < 0.3).astype(np.uint8) * 255
    depth = rng.uniform(H * W, 0.5, 3.0).reshape(H, W).astype(np.float32)
    depth[3, 4] = np.nan; depth[5, 6] = np.inf; depth[7, 8] = 0.0; depth[9, 10] = -1.0; depth[2, 2] = 1e-7
    edges[[3, 5, 7, 9, 2], [4, 6, 8, 10, 2]] = 1
    uv, z = oracle.edge_list(edges, depth, z_min=1e-6)
    keep = (edges != 0) & np.isfinite(depth) & (depth > 1e-6)
    vs, us = np.nonzero(keep)                       # numpy's nonzero is raster (row-major) order
    assert np.array_equal(uv[:, 0], us) and np.array_equal(uv[:, 1], vs)
    assert np.array_equal(z, depth[vs, us])
    # e_max sub-sampling: entries floor(j n / e_max) of the full list (reading S6)
    n = len(z); e_max = 17
    uv2, z2 = oracle.edge_list(edges, depth, z_min=1e-6, e_max=e_max)
    idx = (np.arange(e_max) * n) // e_max
    assert np.array_equal(uv2, uv[idx]) and np.array_equal(z2, z[idx])
    uv3, _ = oracle.edge_list(edges, depth, e_max=10 * n)
    assert len(uv3) == n
    # the DTF uses ALL nonzero edge pixels regardless of depth
    assert oracle.edt(edges)[7, 8] == 0.0


def test_canonical_pairs_is_stable_sort_by_target_then_source():
    rng = SplitMix64(11)
    P = 400
    pairs = np.stack([rng.integers(P, 9), rng.integers(P, 9)], axis=1).astype(np.int32)
    srt, perm = oracle.canonical_pairs(pairs)
    order = np.lexsort((np.arange(P), pairs[:, 0], pairs[:, 1]))   # target major, source, then input index
    assert np.array_equal(perm, order.astype(np.int32))
    assert np.array_equal(srt, pairs[order])
