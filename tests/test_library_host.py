"""CPU-side tests of libqmc.so: it loads, exports every symbol include/qmc.h declares, validates
its inputs, and qmc_plan generates and compiles sector code without a GPU (NVRTC cross-compiles).
No compute entry point is called here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2305_19768_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    from paper_2305_19768_b200 import build, binding
    build.build()
    binding.lib()
    return binding


def test_header_symbols_exported(B):
    header = open(os.path.join(ROOT, "include", "qmc.h")).read()
    declared = set(re.findall(r"\b(qmc_[a-z0-9_]+)\s*\(", header))
    declared -= {"qmc_plan_s"}
    assert declared == set(B.SYMBOLS), declared ^ set(B.SYMBOLS)
    L = C.CDLL(B.LIB_PATH)
    for name in declared:
        assert hasattr(L, name), name


def test_struct_sizes_match_header(B):
    # qmc_sector_desc: 6 + 8 + 2 int32, 4 doubles, 5 pointers; qmc_job: 2 int32 + 9 u64 + 2 doubles
    assert C.sizeof(B.SectorDesc) == 64 + 32 + 40
    assert C.sizeof(B.JobC) == 8 + 72 + 16
    assert C.sizeof(B.PlanOpts) == 48
    # qmc_piece: 4 int32 + 2 u64; qmc_presample_opts: 4 doubles; qmc_presample_info: 3 doubles + 2 int32;
    # qmc_adaptive_opts: 5 doubles + 3 u64 + 4 int32
    assert C.sizeof(B.PieceC) == 32 and C.sizeof(B.PresampleOpts) == 32 and C.sizeof(B.PresampleInfo) == 32
    assert C.sizeof(B.AdaptiveOpts) == 80


def test_math_tables_against_long_double(B):
    """The tables behind the kernels' own log / exp / sincos / atan2 (csrc/qmc_math.cuh), recomputed here
    in numpy long double (x87 extended): every entry is the correctly rounded double (<= 0.51 ulp)."""
    lt, et, tt = B.qmc_debug_math_tables()
    LD = np.longdouble
    ln2 = np.log(LD(2))
    i = np.arange(1025)
    c = lt[0::2]
    assert np.array_equal(c, (LD(1) / (LD(1) + i.astype(LD) / LD(1024))).astype(np.float64))
    L_ref = -np.log(c.astype(LD)) - np.where(i > 424, ln2, LD(0))
    assert np.max(np.abs(lt[1::2].astype(LD) - L_ref)) <= 0.51 * np.spacing(0.35)
    assert np.max(np.abs(lt[1::2])) <= 0.3467                                       # |L_i| <= log(2) / 2: the split at i = 424
    assert lt[1] == 0.0 and lt[2049] == 0.0 and lt[0] == 1.0 and lt[2048] == 0.5   # exact around x = 1
    e_ref = np.exp2(np.arange(256).astype(LD) / LD(256))
    assert np.max(np.abs(et.astype(LD) - e_ref) / e_ref) <= 0.51 * 2.0 ** -52
    ang = LD(2) * np.arctan2(LD(0), LD(-1)) * np.arange(256).astype(LD) / LD(256)
    assert np.max(np.abs(tt[0::2].astype(LD) - np.cos(ang))) <= 0.51 * 2.0 ** -53
    assert np.max(np.abs(tt[1::2].astype(LD) - np.sin(ang))) <= 0.51 * 2.0 ** -53
    assert tt[128] == 0.0 and tt[129] == 1.0 and tt[256] == -1.0 and tt[257] == 0.0


def test_allocate_lattices_matches_the_oracle(B):
    """Eq. (6) through the C ABI against oracle/adaptive.py, which tests/test_oracle_adaptive.py
    pins to the Lagrange conditions; host arithmetic, so this parity test needs no GPU."""
    from oracle import adaptive as A
    rng = np.random.default_rng(21)
    for alpha in (1.0, 2.0, 3.0):
        N = 40
        w = 10.0 ** rng.uniform(-8, 2, N)
        tau = rng.uniform(80, 1500, N)
        c2 = rng.uniform(0.0, 4.0, N)
        w[3] = 0.0
        c2[7] = 0.0
        got = B.qmc_allocate_lattices(w, tau, c2, alpha, 1e-9)
        want = np.array(A.allocate_lattices(w, tau, c2, alpha, 1e-9))
        assert got[3] == 0.0 and got[7] == 0.0
        assert np.allclose(got, want, rtol=1e-13, atol=0)
    for bad in (dict(alpha=0.0), dict(V=0.0), dict(tau=[1.0, -1.0])):
        kw = dict(w=[1.0, 1.0], tau=[1.0, 1.0], c_abs2=[1.0, 1.0], alpha=2.0, V=1.0)
        kw.update(bad)
        with pytest.raises(B.QmcError) as e:
            B.qmc_allocate_lattices(**kw)
        assert e.value.status == B.QMC_ERR_INVALID_ARG


def test_cubin_disk_cache_is_used_by_a_second_process(B, tmp_path):
    """QMC_CUBIN_CACHE=<dir>: the first process compiles and stores, a second one loads the same cubin (its module
    log says so) and generates identical source; without the variable nothing is written."""
    import subprocess
    import sys
    code = ("import sys; sys.path.insert(0, %r)\n"
            "from paper_2305_19768_b200 import binding as B, workloads as W\n"
            "p = B.qmc_plan(W.config_toy().sectors)\n"
            "print(p.module_log(0).strip().splitlines()[-1])\n"
            "print(len(p.module_source(0)))\n" % ROOT)
    env = dict(os.environ, QMC_CUBIN_CACHE=str(tmp_path))
    first = subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, check=True).stdout.splitlines()
    files = sorted(os.listdir(tmp_path))
    assert len(files) == 1 and files[0].startswith("qmc_sm100a_") and files[0].endswith(".cubin")
    assert "loaded from" not in first[0]
    second = subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, check=True).stdout.splitlines()
    assert "loaded from" in second[0] and files[0] in second[0]
    assert second[1] == first[1]
    assert sorted(os.listdir(tmp_path)) == files
    env.pop("QMC_CUBIN_CACHE")
    other = tmp_path / "unused"
    other.mkdir()
    subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, check=True)
    assert os.listdir(other) == []


def test_status_strings(B):
    L = B.lib()
    for code in range(-6, 1):
        assert L.qmc_status_str(code).decode() not in ("", "unknown status")
    assert L.qmc_status_str(-99).decode() == "unknown status"


def test_plan_compiles_every_class_without_gpu(B):
    wl1, wl3 = W.config_euclid(n_sectors=2), W.config_physical(n_sectors=1)
    toy = W.config_toy()
    plan = B.qmc_plan(toy.sectors + wl1.sectors + wl3.sectors, sectors_per_module=2)
    assert plan.J == 3
    assert plan.modules() == 3          # toy (real, d=2), real d=4, deformed d=5
    for i in range(plan.modules()):
        src, log = plan.module_source(i), plan.module_log(i)
        assert "qmc_eval_kernel" in src and "struct Sector_0" in src
        assert "registers" in log and "0 bytes spill stores" in log
    # cost model: a deformed d=5 evaluation is several times a real d=4 one
    assert plan.sector_flops(3) > 4 * plan.sector_flops(1) > 0
    assert plan.sector_ops(1) > 50
    assert plan.workspace_bytes(8, 256) > 0
    plan.destroy()


def test_plan_option_combinations_compile(B):
    """Every compile-time variant of the kernels builds for every class: CUDA-library math (A/B), 64-bit lattice
    indices, one point per thread at one CTA per SM."""
    secs = W.config_toy().sectors + W.config_euclid(n_sectors=1).sectors + W.config_physical(n_sectors=1).sectors
    for opts in ({"libdevice_math": 1}, {"wide_lattice": 1},
                 {"libdevice_math": 1, "wide_lattice": 1, "points_per_thread": 1, "ctas_per_sm": 1}):
        plan = B.qmc_plan(secs, **opts)
        assert plan.modules() == 3
        src = plan.module_source(plan.modules() - 1)
        assert ("#define QMC_LIBDEVICE_MATH 1" in src) == bool(opts.get("libdevice_math"))
        assert ("#define QMC_WIDE 1" in src) == bool(opts.get("wide_lattice"))
        plan.destroy()


def test_plan_source_is_deterministic(B):
    wl = W.config_euclid(n_sectors=1)
    p1, p2 = B.qmc_plan(wl.sectors), B.qmc_plan(wl.sectors)
    assert p1.module_source(0) == p2.module_source(0)
    p1.destroy()
    p2.destroy()


def test_plan_rejects_bad_descriptions(B):
    s = W.config_euclid(n_sectors=1).sectors[0]
    with pytest.raises(B.QmcError) as e:
        B.qmc_plan([])
    assert e.value.status == B.QMC_ERR_INVALID_ARG
    import copy
    bad = copy.deepcopy(s)
    bad.U_coef = bad.U_coef.copy()
    bad.U_coef[1] = np.nan
    with pytest.raises(B.QmcError) as e:
        B.qmc_plan([bad])
    assert e.value.status == B.QMC_ERR_INVALID_ARG
    bad = copy.deepcopy(s)
    bad.transform = 7
    with pytest.raises(B.QmcError) as e:
        B.qmc_plan([bad])
    assert e.value.status == B.QMC_ERR_UNSUPPORTED
    bad = copy.deepcopy(s)
    bad.n_orders = 6                       # more than QMC_MAX_ORDERS = 5
    bad.logc = np.ones(60)
    with pytest.raises(B.QmcError) as e:
        B.qmc_plan([bad])
    assert e.value.status == B.QMC_ERR_INVALID_ARG
    bad = copy.deepcopy(s)
    bad.first_order, bad.n_orders = 3, 3   # degree 5 > QMC_MAX_LOG_DEGREE = 4
    bad.logc = np.ones(60)
    with pytest.raises(B.QmcError) as e:
        B.qmc_plan([bad])
    assert e.value.status == B.QMC_ERR_INVALID_ARG
    with pytest.raises(TypeError):
        B.qmc_plan([s], no_such_option=1)


def test_compute_calls_fail_loudly_without_gpu(B):
    """No CPU fallback: on a box without a CUDA device binding the workspace reports QMC_ERR_CUDA."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    plan = B.qmc_plan(W.config_toy().sectors)
    buf = np.zeros(1 << 20, np.uint8)
    addr = (buf.ctypes.data + 255) // 256 * 256
    rc = B.lib().qmc_plan_bind_workspace(plan.handle, C.c_void_p(addr), 1 << 19)
    assert rc == B.QMC_ERR_CUDA
    assert B.lib().qmc_last_error().decode() != ""
    # every call that would need the device refuses before it, with a status, not a crash
    out = (C.c_int64 * 2)()
    assert B.lib().qmc_plan_slow_path_counts(plan.handle, out, None) == B.QMC_ERR_WORKSPACE
    assert B.lib().qmc_plan_last_job_clocks(plan.handle, out, 1) == B.QMC_ERR_WORKSPACE
    plan.destroy()
    keep = []
    sd = B.marshal_sector(W.config_physical(n_sectors=1).sectors[0], keep)
    info = B.PresampleInfo()
    z = np.ones(8, np.uint64)
    sh = np.full(8, 0.25)
    rc = B.lib().qmc_presample_lambda(C.byref(sd), 101, z.ctypes.data_as(C.c_void_p), sh.ctypes.data_as(C.c_void_p), None,
                                      C.c_void_p(addr), 1 << 19, C.byref(info), None)
    assert rc == B.QMC_ERR_CUDA
    rc = B.lib().qmc_presample_lambda_static(C.byref(sd), 101, z.ctypes.data_as(C.c_void_p), sh.ctypes.data_as(C.c_void_p), None,
                                             C.byref(info), None)
    assert rc == B.QMC_ERR_CUDA


def test_static_presampling_limit_is_checked_before_any_device_call(B):
    """qmc_presample_lambda_static: F beyond QMC_PRESAMPLE_STATIC_MAX_TERMS is refused with QMC_ERR_WORKSPACE and a message
    naming the limit -- with or without a GPU (the check precedes every CUDA call); the array is 96 KiB."""
    import copy
    assert B.lib().qmc_presample_static_max_bytes() == 96 * 1024
    s = W.config_physical(n_sectors=1).sectors[0]
    big = copy.deepcopy(s)
    reps = 1 << int(np.ceil(np.log2(4097.0 / len(s.F_coef))))
    big.F_coef = np.tile(np.asarray(s.F_coef, np.float64) / reps, reps)
    big.F_exp = np.tile(np.asarray(s.F_exp, np.uint8), (reps, 1))
    keep = []
    sd = B.marshal_sector(big, keep)
    assert sd.nF > 4096
    info = B.PresampleInfo()
    z = np.ones(8, np.uint64)
    sh = np.full(8, 0.25)
    rc = B.lib().qmc_presample_lambda_static(C.byref(sd), 101, z.ctypes.data_as(C.c_void_p), sh.ctypes.data_as(C.c_void_p), None,
                                             C.byref(info), None)
    assert rc == B.QMC_ERR_WORKSPACE
    assert "4096" in B.lib().qmc_last_error().decode()


def test_product_does_not_import_oracle():
    """The product path never routes through the oracle (package sources and csrc/ do not name it)."""
    pkg = os.path.join(ROOT, "paper_2305_19768_b200")
    for dirpath, _dirs, files in os.walk(pkg):
        if os.path.basename(dirpath) in ("build", "__pycache__"):
            continue
        for fn in files:
            if not fn.endswith((".py", ".cpp", ".cu", ".cuh", ".h")):
                continue
            text = open(os.path.join(dirpath, fn)).read()
            assert not re.search(r"^\s*(from|import)\s+oracle\b", text, re.M), fn
            assert "qmc_oracle" not in text and "libqmc_oracle" not in text, fn


def test_sector_too_large_for_the_constant_bank_is_refused_clearly(B):
    """A module's sectors keep their coefficients in the 64 KB constant bank next to the math tables
    (csrc/qmc_api.cpp, kConstPoolDoubles*): a single sector with more coefficients than a module can hold is refused
    with QMC_ERR_UNSUPPORTED and a message, instead of failing inside NVRTC / ptxas."""
    rng = np.random.default_rng(3)
    pool = W._exponent_vectors(8, 0, 8)                      # 12 870 monomials of degree <= 8 in 8 variables
    pick = np.sort(rng.choice(len(pool), size=7600, replace=False))
    s = W.draw_euclid_sector(np.random.Generator(np.random.PCG64(1)), 8)
    s.F_exp = np.ascontiguousarray(pool[pick])
    s.F_coef = rng.uniform(0.1, 1.0, size=len(pick))
    with pytest.raises(B.QmcError) as e:
        B.qmc_plan([s])
    assert e.value.status == B.QMC_ERR_UNSUPPORTED and "constant-bank coefficients" in e.value.detail


def test_unpivoted_lu_of_the_deformation_matrix_has_pivots_of_modulus_at_least_one():
    """Reading Q16: the kernel's determinant is an unrolled LU WITHOUT pivoting.  That is safe for every
    input, not just "in practice": M = 1 - i lambda (D H + diag(g)) with D = diag(x_i (1 - x_i)) > 0, H the symmetric
    Hessian of F and g_i = (1 - 2 x_i) dF/dx_i is similar, by the diagonal scaling D^(1/2), to 1 - i lambda S with S
    real symmetric -- a matrix whose Hermitian part is the identity.  Diagonal similarity leaves the pivots unchanged,
    and the Schur complements of a matrix with Hermitian part 1 again have Hermitian part >= 1, so every pivot has
    real part >= 1: no pivot is ever small, the multipliers are bounded by the entries.  Checked here on random
    matrices of exactly that structure (numpy only), including badly scaled D and large lambda |H|."""
    rng = np.random.default_rng(16)
    worst = np.inf
    for trial in range(400):
        d = int(rng.integers(2, 9))
        x = rng.uniform(1e-8, 1.0 - 1e-8, d) if trial % 3 else rng.choice([1e-12, 0.5, 1 - 1e-12], d)
        D = x * (1.0 - x)
        H = rng.standard_normal((d, d)) * 10.0 ** rng.uniform(-2, 4)
        H = H + H.T
        g = (1.0 - 2.0 * x) * rng.standard_normal(d) * 10.0 ** rng.uniform(-2, 4)
        lam = 10.0 ** rng.uniform(-2, 2)
        M = np.eye(d) - 1j * lam * (D[:, None] * H + np.diag(g))
        A = M.copy()
        det = 1.0 + 0.0j
        for c in range(d):                                  # the kernel's elimination order, no row exchanges
            piv = A[c, c]
            worst = min(worst, piv.real)
            det *= piv
            for r in range(c + 1, d):
                f = A[r, c] / piv
                A[r, c + 1:] -= f * A[c, c + 1:]
        ref = np.linalg.det(M)                              # LAPACK, partial pivoting
        assert abs(det - ref) <= 1e-9 * abs(ref), (trial, det, ref)
    assert worst >= 1.0 - 1e-9, worst


def test_log_algorithm_of_the_kernels_emulated_in_exactly_rounded_arithmetic(B):
    """qmc_log_nocheck (csrc/qmc_math.cuh) step by step on the host, every fma / mul / add as the correctly rounded
    value of the exact rational result (Python Fractions), with the table the modules embed: the design -- 1025-entry
    table, |r| <= 2^-11, log1p to r^4 -- is accurate to 3e-16 max(1, |log x|) everywhere and keeps a relative accuracy
    of 1.2e-14 (the dropped term r^5/5 against r) where log x -> 0.  (The GPU per-point parity tests check the compiled function against the oracle.)"""
    import math
    import struct
    from fractions import Fraction as Fr
    lt, _, _ = B.qmc_debug_math_tables()
    ln2_hi = float.fromhex("0x1.62e42fefa39efp-1")
    c2, c3, c4 = -0.5, float.fromhex("0x1.5555555555555p-2"), -0.25
    rnd = lambda q: float(q)                                    # Fraction -> nearest double

    def qlog(x):
        bits = struct.unpack("<Q", struct.pack("<d", x))[0]
        hi, lo = bits >> 32, bits & 0xffffffff
        idx = ((hi & 0xfffff) + 0x200) >> 10
        e = (hi >> 20) - 1023 + (1 if idx > 424 else 0)
        m = struct.unpack("<d", struct.pack("<Q", (((hi & 0xfffff) | 0x3ff00000) << 32) | lo))[0]
        c, L = lt[2 * idx], lt[2 * idx + 1]
        r = rnd(Fr(m) * Fr(c) - 1)
        q = rnd(Fr(r) * Fr(c4) + Fr(c3))
        q = rnd(Fr(r) * Fr(q) + Fr(c2))
        r2 = rnd(Fr(r) * Fr(r))
        base = rnd(Fr(e) * Fr(ln2_hi) + Fr(L))
        p = rnd(Fr(r2) * Fr(q) + Fr(r))
        assert abs(r) <= 2.0 ** -11 * 1.0001
        return rnd(Fr(p) + Fr(base))

    rng = np.random.default_rng(12)
    xs = np.concatenate([rng.uniform(1.0, 2.0, 1500) * 2.0 ** rng.integers(-300, 300, 1500), rng.uniform(0.5, 2.0, 1500),
                         1.0 + rng.uniform(-1, 1, 600) * 10.0 ** rng.uniform(-12, -2, 600), [1.0, 2.0, 0.5, 1.0 + 2.0 ** -52]])
    worst_abs = worst_rel = 0.0
    for x in xs:
        got, ref = qlog(float(x)), np.log(np.longdouble(x))
        err = abs(float(np.longdouble(got) - ref))
        worst_abs = max(worst_abs, err / max(1.0, abs(float(ref))))
        if ref != 0:
            worst_rel = max(worst_rel, err / abs(float(ref)))
    assert qlog(1.0) == 0.0
    assert worst_abs <= 3e-16 and worst_rel <= 1.2e-14, (worst_abs, worst_rel)
