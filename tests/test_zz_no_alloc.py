"""epo_edt_no_alloc against the library's ordinary distance-transform path (epo_set_views -> epo_get_dtf).

The entry point exists for programs that cannot let a library allocate device memory: a server or trainer whose own
allocator already holds all of HBM (a cudaMalloc behind its back fails or starves it), and per-frame loops where the
device-wide stall of cudaMalloc / cudaFree is not affordable.  Its only work buffer is a 2 MiB array built into
libepo.so, shared by every call on a GPU and never cleared, so what has to be shown is that (1) it returns exactly the
field the allocating path returns (the distance transform is integer work: the suite's tolerance for it is bit
equality), (2) a second call right after the first is not disturbed by what the first one left in that buffer --
different image, different size, in both orders -- and (3) an image beyond the built-in limit is refused with a
message instead of overrunning the array.

This file sorts last on purpose (`pytest --collect-only`): under `pytest -x` a failure here hides nothing after it.
It keeps no state between tests and needs none from the other files, so it passes alone in a fresh process as well as
at the end of the whole suite.
"""
import numpy as np
import pytest

from epo_scenes import SplitMix64, make_scene

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _need_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2607_00579_b200 import build
    build.build()


def _reference_fields(edges, W, H):
    """fp32 fields of the edge maps [N][H][W] through the existing, allocating path."""
    import torch
    from paper_2607_00579_b200 import Epo, epo_config_default
    N = edges.shape[0]
    K = np.tile(np.array([300.0, 300.0, W / 2, H / 2], np.float32), (N, 1))
    poses = np.tile(np.eye(4, dtype=np.float32)[:3].reshape(1, 12), (N, 1))
    depth = np.ones((N, H, W), np.float32)
    e = Epo(epo_config_default(n_views=N, width=W, height=H, stream=torch.cuda.current_stream().cuda_stream))
    e.set_views(K, poses, depth, np.ascontiguousarray(edges))
    out = np.stack([e.get_dtf(i) for i in range(N)])
    e.destroy()
    return out


def _masks(N, H, W, seed):
    rng = SplitMix64(seed)
    m = np.zeros((N, H, W), np.uint8)
    m[0] = rng.uniform(H * W).reshape(H, W) < 0.03          # the paper's edge density, roughly
    m[1, H // 3, (2 * W) // 3] = 255                          # a single pixel: the longest searches
    if N > 2:
        m[2] = 0                                              # no edge at all: the sentinel W + H everywhere
    if N > 3:
        m[3, 5, :] = 1                                        # one full row: every other row holds the row-pass sentinel
    return m


def test_two_calls_in_a_row_match_the_allocating_path():
    import torch
    from paper_2607_00579_b200 import edt_no_alloc
    big = dict(W=518, H=392)                                  # the paper's frame, 39 % of the built-in buffer
    small = dict(W=45, H=37)                                  # ragged: neither a multiple of 32 nor of 8
    mb, ms = _masks(4, big["H"], big["W"], 11), _masks(4, small["H"], small["W"], 12)
    rb, rs = _reference_fields(mb, **big), _reference_fields(ms, **small)
    stream = torch.cuda.current_stream().cuda_stream
    # caller-owned inputs and outputs, made before the calls under test; outputs pre-filled with NaN so that an
    # unwritten pixel cannot pass
    db, ds = torch.from_numpy(mb).cuda(), torch.from_numpy(ms).cuda()
    ob = torch.full((4, big["H"], big["W"]), float("nan"), device="cuda")
    os_ = torch.full((4, small["H"], small["W"]), float("nan"), device="cuda")
    edt_no_alloc(db[0], ob[0], stream)                        # first call on this device: resolves the array's address
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    # back to back on one stream, sizes alternating, so that every call finds the previous call's rows in the buffer
    order = [(db, ob, 1), (ds, os_, 0), (db, ob, 2), (ds, os_, 1), (ds, os_, 2), (db, ob, 3), (ds, os_, 3), (db, ob, 0)]
    for d, o, i in order:
        edt_no_alloc(d[i], o[i], stream)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before        # the calls took no device memory
    assert np.array_equal(ob.cpu().numpy(), rb)
    assert np.array_equal(os_.cpu().numpy(), rs)
    assert rs[2].min() == small["W"] + small["H"] and rb[2].max() == big["W"] + big["H"]   # the empty view


def test_same_image_twice_gives_the_same_bits_and_sizes_beyond_the_limit_are_refused():
    import torch
    from paper_2607_00579_b200 import EDT_NO_ALLOC_MAX_PIXELS, EPO_ERR_INVALID_ARG, EPO_ERR_UNSUPPORTED, EpoError, edt_no_alloc
    sc = make_scene(1)                                        # the Tiny configuration's own edge maps
    d = torch.from_numpy(np.ascontiguousarray(sc.edges)).cuda()
    ref = _reference_fields(sc.edges, sc.W, sc.H)
    a = torch.empty((sc.H, sc.W), device="cuda"); b = torch.empty_like(a)
    edt_no_alloc(d[0], a)
    edt_no_alloc(d[0], b)
    torch.cuda.synchronize()
    assert np.array_equal(a.cpu().numpy(), ref[0]) and np.array_equal(b.cpu().numpy(), ref[0])
    # exactly at the limit: accepted; one row more: refused before anything is launched, output untouched
    W = 1024; H = EDT_NO_ALLOC_MAX_PIXELS // W
    edges = torch.zeros((H + 1, W), dtype=torch.uint8, device="cuda"); edges[7, 9] = 1
    out = torch.full((H + 1, W), -1.0, device="cuda")
    edt_no_alloc(edges[:H], out[:H])
    torch.cuda.synchronize()
    yy, xx = np.mgrid[0:H, 0:W]
    want = np.sqrt(((yy - 7) ** 2 + (xx - 9) ** 2).astype(np.float64)).astype(np.float32)   # one edge pixel: the closed form
    assert np.array_equal(out[:H].cpu().numpy(), want) and float(out[H].max()) == -1.0
    out.fill_(-1.0)
    with pytest.raises(EpoError) as ei:
        edt_no_alloc(edges, out)
    assert ei.value.status == EPO_ERR_UNSUPPORTED and "EPO_EDT_NO_ALLOC_MAX_PIXELS" in str(ei.value)
    torch.cuda.synchronize()
    assert float(out.max()) == -1.0
    with pytest.raises(EpoError) as ei:                       # a host array is not a device pointer
        edt_no_alloc(np.zeros((8, 8), np.uint8), out[:8, :8].contiguous())
    assert ei.value.status == EPO_ERR_INVALID_ARG
