"""Host-side checks of the C-ABI library that need no GPU: it loads, exports every symbol that
include/epo.h declares, validates arguments, and fails loudly without a CUDA device (no CPU fallback)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    from paper_2607_00579_b200 import build
    build.build()
    import paper_2607_00579_b200 as pkg
    return pkg.lib()


def test_exports_every_declared_symbol(L):
    import paper_2607_00579_b200 as pkg
    header = open(os.path.join(ROOT, "include", "epo.h")).read()
    declared = set(re.findall(r"EPO_API\s+[\w\s\*]+?\b(epo_\w+)\s*\(", header))
    assert declared == set(pkg.SYMBOLS), declared ^ set(pkg.SYMBOLS)
    for name in declared:
        assert hasattr(L, name), name
    assert b"sm_100a" in L.epo_version()


def test_config_defaults_are_the_papers(L):
    import paper_2607_00579_b200 as pkg
    cfg = pkg.epo_config_default()
    assert (cfg.clamp_start, cfg.clamp_end, cfg.clamp_steps) == (10.0, 6.0, 1000)
    assert abs(cfg.lr_max - 3e-3) < 1e-9 and (cfg.warmup_steps, cfg.max_steps) == (25, 2000)
    assert abs(cfg.beta1 - 0.9) < 1e-7 and abs(cfg.beta2 - 0.999) < 1e-7
    assert (cfg.w1, cfg.w2) == (25, 50) and abs(cfg.eps1 - 0.5) < 1e-7 and abs(cfg.eps2 - 0.1) < 1e-7
    assert cfg.huber_delta == 1.0 and cfg.smooth_window == 1
    assert pkg.lib().epo_config_default(None) == pkg.EPO_ERR_INVALID_ARG


def test_create_rejects_bad_configs_without_touching_cuda(L):
    import paper_2607_00579_b200 as pkg
    for bad in (dict(n_views=1, width=64, height=64), dict(n_views=4, width=1, height=64),
                dict(n_views=4, width=64, height=70000), dict(n_views=4, width=64, height=64, huber_delta=0.0),
                dict(n_views=4, width=64, height=64, dtf_format=7), dict(n_views=4, width=64, height=64, max_steps=10)):
        cfg = pkg.epo_config_default(**bad)
        h = C.c_void_p()
        assert L.epo_create(C.byref(cfg), C.byref(h)) == pkg.EPO_ERR_INVALID_ARG
        assert not h
    assert L.epo_create(None, None) == pkg.EPO_ERR_INVALID_ARG
    L.epo_destroy(None)   # NULL-safe
    assert L.epo_step(None, 1, None, None) == pkg.EPO_ERR_INVALID_ARG
    assert L.epo_last_error(None) == b"null context"


def test_fails_loudly_without_a_gpu(L):
    """The product path has no CPU fallback: on a box without CUDA epo_create returns EPO_ERR_CUDA."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    import paper_2607_00579_b200 as pkg
    cfg = pkg.epo_config_default(n_views=4, width=64, height=48)
    with pytest.raises(pkg.EpoError) as ei:
        pkg.Epo(cfg)
    assert ei.value.status == pkg.EPO_ERR_CUDA


def test_product_package_never_touches_the_oracle():
    """Neither side imports or links the other (independence of oracle and CUDA path)."""
    pkg_dir = os.path.join(ROOT, "paper_2607_00579_b200")
    for dirpath, _, files in os.walk(pkg_dir):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh", ".cpp")):
                src = open(os.path.join(dirpath, f), errors="ignore").read()
                assert "oracle" not in src.lower().replace("no cpu fallback", ""), os.path.join(dirpath, f)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2607_00579_b200" not in src and "libepo" not in src and "epo.h" not in src
