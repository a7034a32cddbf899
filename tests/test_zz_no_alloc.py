"""qmc_presample_lambda_static: the entry point that allocates nothing (device scratch = a 96 KiB file-scope __device__
array inside libqmc.so, host side on the stack; include/qmc.h) against the existing path qmc_presample_lambda with
caller-provided scratch.  Both launch the same kernel on the same inputs: the selected lambda, the step count and the
ok flag are equal, max Im F / min |F| agree to the tolerance the presampling tests use (tests/test_gpu_physical.py).

The array is shared by all calls and keeps the last call's contents, so the calls below come in a row with DIFFERENT
sectors, candidate counts and dimensions: a counter or key that was not reset would show in the second result.
This file is named to be collected last (the suite runs with pytest -x); it passes alone in a fresh process too.
"""
import copy

import numpy as np
import pytest

from paper_2305_19768_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device; there is no CPU fallback"
    torch.cuda.set_device(0)
    return torch


@pytest.fixture(scope="module")
def B():
    from paper_2305_19768_b200 import build, binding
    build.build()
    binding.lib()
    return binding


def _same(got, want):
    assert (got["ok"], got["lam"], got["steps"]) == (want["ok"], want["lam"], want["steps"]), (got, want)
    for key in ("max_im_f", "min_abs_f"):
        if np.isnan(want[key]):
            assert np.isnan(got[key]), (key, got, want)
        else:
            assert got[key] == pytest.approx(want[key], rel=1e-12, abs=0.0), (key, got, want)


def _cases():
    """(sector, n_pre, z, shift, opts): BASELINE.json config 3 sectors (d = 5, 18 monomials) and the d = 1 sectors of
    pins P15 / P19, with option sets that end in ok = 1, in the fallback (ok = 0, distance unreachable) and in
    lambda_min (nothing passes the sign check)."""
    from tests.test_oracle_pins_physical import physical_1d_sector
    from tests.test_oracle_pins_transforms import _cubic_sector
    rng = np.random.Generator(np.random.PCG64(77))
    out = []
    for s in W.config_physical(n_sectors=3).sectors:
        out.append((s, 4099, W.draw_z(rng, 4099, 5), W.draw_shifts(rng, 1, 5)[0], dict(min_abs_f=0.02)))
    one = np.array([1], np.uint64)
    out.append((_cubic_sector(0.4, -4.0), 20011, one, np.array([0.123]), dict(lambda_max=2.0, decrease=0.9)))
    s1 = physical_1d_sector(0.37, -0.5, 0.5, -1e-12, W.TRANSFORM_BAKER)
    out.append((s1, 1009, one, np.array([0.3]), dict(min_abs_f=0.5, lambda_min=0.3)))           # few candidates, fallback
    out.append((physical_1d_sector(0.37, -0.5, 0.5, +0.3, W.TRANSFORM_BAKER), 101, one, np.array([0.3]),
                dict(lambda_min=0.05)))                                                           # no candidate passes
    out.append((_cubic_sector(0.4, -4.0, transform=133), 4099, one, np.array([0.71]), dict(lambda_max=2.0, decrease=0.8)))
    return out


def test_static_scratch_entry_point_matches_the_caller_scratch_path(torch_cuda, B):
    assert B.lib().qmc_presample_static_max_bytes() == 96 * 1024
    cases = _cases()
    want = [B.qmc_presample_lambda(s, n, z, sh, **o) for s, n, z, sh, o in cases]
    seen = set()
    for rnd in range(2):                                    # two passes: every case also runs after every other one
        for (s, n, z, sh, o), w in zip(cases, want):
            _same(B.qmc_presample_lambda_static(s, n, z, sh, **o), w)
            seen.add((w["ok"], np.isnan(w["max_im_f"])))
        cases, want = cases[::-1], want[::-1]
    assert seen == {(True, False), (False, False), (False, True)}     # admissible, fallback and lambda_min all occurred
    # the same call twice in a row, and on a side stream
    s, n, z, sh, o = cases[0]
    a = B.qmc_presample_lambda_static(s, n, z, sh, **o)
    b = B.qmc_presample_lambda_static(s, n, z, sh, **o)
    _same(b, a)
    st = torch_cuda.cuda.Stream()
    torch_cuda.cuda.synchronize()
    _same(B.qmc_presample_lambda_static(cases[3][0], cases[3][1], cases[3][2], cases[3][3], stream=st, **cases[3][4]), want[3])


def test_static_scratch_entry_point_allocates_no_device_memory(torch_cuda, B):
    """Free device memory (cudaMemGetInfo) is the same before and after the calls once the array's module is loaded."""
    s, n, z, sh, o = _cases()[0]
    B.qmc_presample_lambda_static(s, n, z, sh, **o)          # set-up: symbol address, lazy module load
    torch_cuda.cuda.synchronize()
    free0, _ = torch_cuda.cuda.mem_get_info()
    for _ in range(5):
        B.qmc_presample_lambda_static(s, n, z, sh, **o)
    torch_cuda.cuda.synchronize()
    free1, _ = torch_cuda.cuda.mem_get_info()
    assert free1 == free0


def test_static_scratch_entry_point_refuses_sizes_beyond_its_maximum(torch_cuda, B):
    """More than QMC_PRESAMPLE_STATIC_MAX_TERMS monomials in F: QMC_ERR_WORKSPACE with a message naming the limit, while
    the caller-scratch path takes the same sector; the refusal leaves the array usable."""
    base = _cases()[0]
    s = base[0]
    big = copy.deepcopy(s)
    reps = 1 << int(np.ceil(np.log2(4097.0 / len(s.F_coef))))  # 18 monomials x 256 = 4608; dividing by 2^k is exact
    big.F_coef = np.tile(np.asarray(s.F_coef, np.float64) / reps, reps)    # the same polynomial, written out longer
    big.F_exp = np.tile(np.asarray(s.F_exp, np.uint8), (reps, 1))
    assert len(big.F_coef) > 4096
    with pytest.raises(B.QmcError) as ei:
        B.qmc_presample_lambda_static(big, base[1], base[2], base[3], **base[4])
    assert "4096" in str(ei.value) and ei.value.status == B.QMC_ERR_WORKSPACE
    r = B.qmc_presample_lambda(big, base[1], base[2], base[3], **base[4])     # the existing path takes it
    w = B.qmc_presample_lambda(s, base[1], base[2], base[3], **base[4])
    assert 0.0 < r["lam"] <= 1.0 and abs(r["steps"] - w["steps"]) <= 1       # same F up to the rounding of the longer sum
    _same(B.qmc_presample_lambda_static(s, base[1], base[2], base[3], **base[4]), w)
