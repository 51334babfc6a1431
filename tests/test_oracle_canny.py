"""Pins of the oracle's Canny edge extraction ("the Canny edge detector [4]"; Alg. 1 l.6,
PAPER.md:374-376; readings C1-C6 in DESIGN.md).  The linear stages are checked against scipy.ndimage (an independent
library routine), the decisions against hand-made gradient fields and step images whose answer is known."""
import numpy as np
import scipy.ndimage as ndi

import oracle


def test_K1_blur_and_sobel_match_scipy():
    rng = np.random.default_rng(5)
    img = rng.integers(0, 256, (37, 53), dtype=np.uint8)
    w = np.array([1, 4, 6, 4, 1], np.int64)
    acc = ndi.correlate(img.astype(np.int64), np.outer(w, w), mode="nearest")
    assert np.array_equal(oracle.canny_blur(img), ((acc + 128) >> 8).astype(np.uint8))
    b = oracle.canny_blur(img)
    kx = np.array([[-1, 0, 1], [-2, 0, 2], [-1, 0, 1]], np.int64)
    gx, gy = oracle.canny_sobel(b)
    assert np.array_equal(gx, ndi.correlate(b.astype(np.int64), kx, mode="nearest"))
    assert np.array_equal(gy, ndi.correlate(b.astype(np.int64), kx.T, mode="nearest"))
    assert np.array_equal(oracle.canny_blur(np.full((9, 9), 77, np.uint8)), np.full((9, 9), 77, np.uint8))   # weights sum to 256


def test_K2_step_images():
    """A vertical / horizontal step gives one straight, one-pixel-wide line next to the step on every interior row /
    column (of the two equally strong columns the first stays); a constant image gives nothing."""
    img = np.zeros((40, 60), np.uint8); img[:, 30:] = 200
    e = oracle.canny(img, 50, 100)
    assert e[1:-1, 29].all() and e.sum() == 38 and not e[0].any() and not e[-1].any()
    eh = oracle.canny(np.ascontiguousarray(img.T), 50, 100)
    assert eh[29, 1:-1].all() and eh.sum() == 38
    assert oracle.canny(np.full((20, 20), 123, np.uint8), 1, 2).sum() == 0
    # a diagonal step: a connected, thin staircase -- one or two pixels per interior row, never a 2x2 block
    yy, xx = np.mgrid[0:50, 0:50]
    d = oracle.canny((200 * (xx > yy)).astype(np.uint8), 50, 100)
    rows = d[3:-3].sum(axis=1)
    assert rows.min() >= 1 and rows.max() <= 2
    assert not (d[:-1, :-1] & d[1:, :-1] & d[:-1, 1:] & d[1:, 1:]).any()
    lab, n = ndi.label(d, structure=np.ones((3, 3)))
    assert n == 1


def _field(H=9, W=12):
    return np.zeros((H, W), np.int32), np.zeros((H, W), np.int32)


def test_K3_thresholds_are_strict_and_compared_squared():
    gx, gy = _field()
    gy[4, 2] = 100; gy[4, 5] = 101; gy[4, 8] = 50; gy[4, 10] = 51     # isolated ridge pixels (vertical gradient)
    c = oracle.canny_suppress(gx, gy, 50, 100)
    assert c[4, 2] == 1 and c[4, 5] == 2 and c[4, 8] == 0 and c[4, 10] == 1 and c.sum() == 4
    gx2, gy2 = _field(); gx2[4, 5] = 60; gy2[4, 5] = 80               # |g| = 100 exactly: not strong
    assert oracle.canny_suppress(gx2, gy2, 50, 100)[4, 5] == 1
    gx2[4, 5] = 61
    assert oracle.canny_suppress(gx2, gy2, 50, 100)[4, 5] == 2


def test_K4_direction_sectors_and_tie_rule():
    """(100, 41) is in the horizontal sector (41/100 < tan 22.5), (100, 42) in the diagonal one: a stronger LEFT
    neighbour suppresses the first only, a stronger upper-left neighbour the second only."""
    for gyv, left_kills, diag_kills in ((41, True, False), (42, False, True)):
        for which in ("left", "diag"):
            gx, gy = _field()
            gx[4, 5] = 100; gy[4, 5] = gyv
            if which == "left": gx[4, 4] = 200
            else: gx[3, 4] = 200
            kept = oracle.canny_suppress(gx, gy, 10, 1000)[4, 5] == 1
            assert kept == (not (left_kills if which == "left" else diag_kills)), (gyv, which)
    gx, gy = _field(); gx[4, 5] = gx[4, 6] = 100                      # two equal neighbours along x: the first stays
    c = oracle.canny_suppress(gx, gy, 10, 1000)
    assert c[4, 5] == 1 and c[4, 6] == 0
    gx, gy = _field(); gx[4, 0] = gx[0, 5] = gx[8, 5] = gx[4, 11] = 500   # border pixels are never candidates
    assert oracle.canny_suppress(gx, gy, 10, 100).sum() == 0
    gx, gy = _field(); gx[4, 5] = 100; gy[4, 5] = -100; gx[3, 6] = 300    # opposite signs: the other diagonal
    assert oracle.canny_suppress(gx, gy, 10, 1000)[4, 5] == 0
    gx[3, 6] = 0; gx[3, 4] = 300
    assert oracle.canny_suppress(gx, gy, 10, 1000)[4, 5] == 1


def test_K5_hysteresis_keeps_what_touches_a_strong_pixel():
    c = np.zeros((10, 16), np.uint8)
    c[2, 1:8] = 1; c[2, 4] = 2            # a weak run with one strong pixel: all kept
    c[5, 1:6] = 1                         # an isolated weak run: dropped
    c[7, 10] = 2; c[8, 11] = 1; c[7, 12] = 1; c[6, 13] = 1   # diagonal chain: 8-connectivity
    c[9, 15] = 1
    e = oracle.canny_hysteresis(c)
    want = np.zeros_like(c); want[2, 1:8] = 1; want[7, 10] = want[8, 11] = want[7, 12] = want[6, 13] = 1
    assert np.array_equal(e, want)
    lab, n = ndi.label(c > 0, structure=np.ones((3, 3)))             # the definition, by connected components
    keep = np.isin(lab, np.unique(lab[c == 2])) & (c > 0)
    assert np.array_equal(e.astype(bool), keep)
    rng = np.random.default_rng(1)
    r = rng.choice([0, 0, 0, 1, 1, 2], size=(64, 80), p=None).astype(np.uint8)
    lab, n = ndi.label(r > 0, structure=np.ones((3, 3)))
    assert np.array_equal(oracle.canny_hysteresis(r).astype(bool), np.isin(lab, np.unique(lab[r == 2])) & (r > 0))


def test_K6_rgb_to_grey_is_bt601_luma_in_fixed_point():
    """Reading C7: grey pixels keep their value exactly; the primaries map to (77, 149, 29) and white to 255 (hand-computed:
    (77 x 255 + 128) >> 8 = 77, (150 x 255 + 128) >> 8 = 149, (29 x 255 + 128) >> 8 = 29); random colours are within one
    grey level of the real-valued luma 0.299 R + 0.587 G + 0.114 B."""
    g = np.arange(256, dtype=np.uint8)
    assert np.array_equal(oracle.rgb_to_grey(np.stack([g, g, g], axis=-1)), g)
    prim = np.array([[255, 0, 0], [0, 255, 0], [0, 0, 255], [255, 255, 255], [0, 0, 0]], np.uint8)
    assert oracle.rgb_to_grey(prim).tolist() == [77, 149, 29, 255, 0]
    rng = np.random.default_rng(5)
    rgb = rng.integers(0, 256, size=(37, 41, 3), dtype=np.uint8)
    y = 0.299 * rgb[..., 0] + 0.587 * rgb[..., 1] + 0.114 * rgb[..., 2]
    assert np.max(np.abs(oracle.rgb_to_grey(rgb).astype(np.float64) - y)) <= 1.0
