"""Host-side checks that need no GPU: the C-ABI library builds, loads and exports every symbol
include/ra_mppi.h declares; struct layouts agree; invalid configs are rejected before any
CUDA call; the product path does not fall back to the CPU."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2209_12842_b200 import binding as B
from paper_2209_12842_b200 import build as cuda_build
from paper_2209_12842_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    cuda_build.build()
    return B.load()


def test_every_declared_symbol_is_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "ra_mppi.h")).read()
    declared = set(re.findall(r"\b(ra_mppi_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(B.EXPORTS), declared ^ set(B.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name


def test_struct_size_is_checked(lib):
    p = W.config0()
    cfg = B.make_config(p)
    env, keep = B.make_env(p)
    cfg.struct_size += 4
    with pytest.raises(B.RaMppiError) as e:
        B.ra_mppi_create(cfg, env)
    assert e.value.status == B.RA_EINVAL


@pytest.mark.parametrize("field,value", [
    ("K", 0), ("M", -1), ("T", 0), ("dt", 0.0), ("alpha", 0.0), ("alpha", 1.0), ("lam", 0.0),
    ("gamma", -1.0), ("eta", 1.0), ("B", 0.0), ("dyn", 7), ("risk", 5), ("nominal", 3), ("noise_kind", 9),
])
def test_invalid_config_is_einval(lib, field, value):
    p = W.config0()
    cfg = B.make_config(p)
    env, keep = B.make_env(p)
    setattr(cfg, field, value)
    with pytest.raises(B.RaMppiError) as e:
        B.ra_mppi_create(cfg, env)
    assert e.value.status == B.RA_EINVAL


def test_create_says_why_it_failed(lib):
    """A caller behind the C ABI gets the reason, not just a status code: ra_mppi_create_error, per calling thread."""
    p = W.config0()
    cfg, (env, keep) = B.make_config(p), B.make_env(p)
    cfg.alpha = 1.5
    ctx = C.c_void_p()
    assert lib.ra_mppi_create(C.byref(cfg), C.byref(env), C.byref(ctx)) == B.RA_EINVAL and not ctx.value
    assert b"alpha" in lib.ra_mppi_create_error()
    with pytest.raises(B.RaMppiError) as e:
        B.ra_mppi_create(cfg, env)
    assert "alpha" in str(e.value)
    cfg = B.make_config(p)
    cfg.M = 513
    with pytest.raises(B.RaMppiError) as e:
        B.ra_mppi_create(cfg, env)
    assert e.value.status == B.RA_EUNSUPPORTED and "M" in str(e.value).replace("RA_EUNSUPPORTED", "").replace("ra_mppi", "")
    import torch
    if not torch.cuda.is_available():
        with pytest.raises(B.RaMppiError) as e:
            B.ra_mppi_create(B.make_config(p), env)
        assert "no CUDA device" in str(e.value) and "no CPU fallback" in str(e.value)


def test_unsupported_sizes(lib):
    p = W.config0()
    for field, value in (("M", 513), ("T", 129)):
        cfg = B.make_config(p)
        env, keep = B.make_env(p)
        setattr(cfg, field, value)
        with pytest.raises(B.RaMppiError) as e:
            B.ra_mppi_create(cfg, env)
        assert e.value.status == B.RA_EUNSUPPORTED


def test_missing_environment_is_einval(lib):
    p = W.config0()
    env, keep = B.make_env(p)
    env.circles = None   # n_circles > 0 without the array (n_circles = 0 alone is a legal empty scene)
    with pytest.raises(B.RaMppiError) as e:
        B.ra_mppi_create(B.make_config(p), env)
    assert e.value.status == B.RA_EINVAL
    p3 = W.config3(K=8).replace(costmap=None)
    with pytest.raises(B.RaMppiError) as e:
        B.ra_mppi_create(B.make_config(p3), B.make_env(p3)[0])
    assert e.value.status == B.RA_EINVAL


def test_null_context_and_destroy_null(lib):
    assert lib.ra_mppi_destroy(None) == B.RA_OK
    assert lib.ra_mppi_step(None, None, None, 0, None) == B.RA_EINVAL
    assert lib.ra_mppi_launches_per_step(None) == 0


def test_no_cpu_fallback_without_gpu(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    p = W.config0()
    with pytest.raises(B.RaMppiError) as e:   # valid config, but no device: must fail loudly
        B.ra_mppi_create(B.make_config(p), B.make_env(p)[0])
    assert e.value.status == B.RA_ECUDA
    from paper_2209_12842_b200.controller import RaMppi
    with pytest.raises(B.RaMppiError):
        RaMppi(p)


def test_product_does_not_import_oracle():
    """The product path never routes through the oracle, and the oracle never uses the product."""
    pat = re.compile(r"(^\s*(import|from)\s+oracle\b)|(#include\s*[<\"].*oracle)|(libra_mppi_oracle)|(oracle[./])", re.M)
    pkg = os.path.join(ROOT, "paper_2209_12842_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                if f == "workloads.py":   # mentions the folder in prose only
                    src = src.replace("``oracle/``", "")
                assert not pat.search(src), f
    pat2 = re.compile(r"(^\s*(import|from)\s+paper_2209_12842_b200)|(#include\s*[<\"].*(ra_mppi\.h|\.cuh))|(libra_mppi\.so)", re.M)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".h")):
            assert not pat2.search(open(os.path.join(ROOT, "oracle", f)).read()), f


def test_tail_and_mean_counts_survive_fp32_parameters(lib):
    """k_tail = ceil((1-alpha) M) and K0 = ceil((1-eta) K) are integer decisions taken from fp32 parameters: the
    library (2^-23 n guard) must agree with the fp64 oracle (1e-9 guard) for every decimal a caller would type,
    including those whose fp32 rounding falls on the wrong side of an integer (G11)."""
    import math

    from oracle import oracle as O
    p = W.config0()
    for M in (1, 2, 10, 16, 20, 37, 64, 100, 128, 256, 300, 512):
        for alpha in (0.01, 0.05, 0.1, 0.25, 0.3, 0.35, 0.5, 0.6, 0.7, 0.75, 0.8, 0.85, 0.9, 0.95, 0.975, 0.99, 0.999):
            k_tail, _ = B.ra_mppi_query_counts(B.make_config(p.replace(M=M, alpha=alpha)))
            assert k_tail == O.tail_count(alpha, M), (alpha, M)
    assert B.ra_mppi_query_counts(B.make_config(p.replace(M=10, alpha=0.7)))[0] == 3       # 0.7f -> 3.0000001
    assert B.ra_mppi_query_counts(B.make_config(p.replace(M=300, alpha=0.9)))[0] == 30     # the paper's N = 300
    # alpha on both sides of an integer (1-alpha) M, 2e-4 away: outside the 2^-23 M = 6e-5 guard window at M = 512
    for k in (1, 13, 26, 400):
        lo, hi = 1.0 - (k - 2e-4) / 512.0, 1.0 - (k + 2e-4) / 512.0
        assert B.ra_mppi_query_counts(B.make_config(p.replace(M=512, alpha=lo)))[0] == k == O.tail_count(lo, 512)
        assert B.ra_mppi_query_counts(B.make_config(p.replace(M=512, alpha=hi)))[0] == k + 1 == O.tail_count(hi, 512)
    for K in (10, 96, 1000, 1024, 4096, 65536):
        for eta in (0.0, 0.05, 0.1, 0.2, 0.25, 0.3, 0.35, 0.5, 0.65, 0.7, 0.8, 0.9, 0.95):
            _, K0 = B.ra_mppi_query_counts(B.make_config(p.replace(K=K, eta=eta)))
            assert K0 == math.ceil((1.0 - eta) * K - 1e-9), (eta, K)
    assert B.ra_mppi_query_counts(B.make_config(p.replace(K=1000, eta=0.7)))[1] == 300
    assert B.ra_mppi_query_counts(B.make_config(p.replace(K=10, eta=0.9)))[1] == 1
    # sharded: the split is taken on the global sample count
    assert B.ra_mppi_query_counts(B.make_config(p.replace(K=100, K_total=1000, k_offset=200, eta=0.35)))[1] == 650
    cfg = B.make_config(p)
    cfg.alpha = 1.0
    with pytest.raises(B.RaMppiError):
        B.ra_mppi_query_counts(cfg)
