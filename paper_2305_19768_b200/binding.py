"""Thin Python binding of ``libqmc.so`` (C ABI: ``include/qmc.h``) -- argument marshalling only.

Same names as the C entry points: :func:`qmc_plan`, :func:`qmc_integrate_sectors`,
:func:`qmc_median_rule`, :func:`qmc_median_integrate_sectors`, the two debug hooks and
:func:`qmc_measure_fp64_peak`.  Every step of the path (lattice points, transforms, integrands,
reductions, median selection, amplitude) runs in the CUDA kernels behind the library; PyTorch is
used for device memory and streams only.  There is no CPU fallback: if ``libqmc.so`` has not
been built (``python -m paper_2305_19768_b200.build``) loading raises, and without a CUDA
device every compute call raises :class:`QmcError`.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

from . import workloads as W

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libqmc.so")
MAXD = 8

QMC_OK = 0
QMC_ERR_INVALID_ARG = -1
QMC_ERR_UNSUPPORTED = -2
QMC_ERR_CUDA = -3
QMC_ERR_WORKSPACE = -4
QMC_ERR_NOT_UNIT = -5
QMC_ERR_COMPILE = -6

# every symbol include/qmc.h declares (tests check that the library exports each one)
SYMBOLS = (
    "qmc_plan", "qmc_plan_orders", "qmc_plan_modules", "qmc_plan_module_source", "qmc_plan_module_log",
    "qmc_plan_sector_flops", "qmc_plan_sector_ops", "qmc_plan_workspace_bytes", "qmc_plan_bind_workspace",
    "qmc_integrate_sectors", "qmc_median_rule", "qmc_median_integrate_sectors", "qmc_debug_lattice_coords",
    "qmc_debug_eval_points", "qmc_debug_math_tables", "qmc_measure_fp64_peak", "qmc_measure_fp64_peak_mixed",
    "qmc_allocate_lattices", "qmc_adaptive_scratch_bytes", "qmc_adaptive_integrate", "qmc_plan_sector_emitted_flops", "qmc_plan_last_stats", "qmc_plan_last_eval_ms", "qmc_plan_slow_path_counts", "qmc_plan_last_job_clocks", "qmc_presample_scratch_bytes", "qmc_presample_lambda", "qmc_presample_static_max_bytes", "qmc_presample_lambda_static", "qmc_integrate_pieces", "qmc_finalize_pieces", "qmc_median_select_pieces",
    "qmc_plan_destroy", "qmc_status_str", "qmc_last_error",
)


class QmcError(RuntimeError):
    def __init__(self, status: int, detail: str):
        super().__init__("libqmc: %s (%d): %s" % (_status_str(status), status, detail))
        self.status = status
        self.detail = detail


class SectorDesc(C.Structure):      # qmc_sector_desc
    _fields_ = [
        ("kind", C.c_int32), ("dim", C.c_int32), ("transform", C.c_int32), ("deformed", C.c_int32),
        ("first_order", C.c_int32), ("n_orders", C.c_int32),
        ("a", C.c_int32 * MAXD),
        ("nU", C.c_int32), ("nF", C.c_int32),
        ("p", C.c_double), ("q", C.c_double), ("lam", C.c_double), ("f_im", C.c_double),
        ("U_coef", C.c_void_p), ("U_exp", C.c_void_p), ("F_coef", C.c_void_p), ("F_exp", C.c_void_p),
        ("logc", C.c_void_p),
    ]


class PlanOpts(C.Structure):        # qmc_plan_opts
    _fields_ = [
        ("validate", C.c_int32), ("threads_per_block", C.c_int32), ("ctas_per_sm", C.c_int32),
        ("max_tiles", C.c_int32), ("sectors_per_module", C.c_int32), ("compile_threads", C.c_int32),
        ("libdevice_math", C.c_int32), ("points_per_thread", C.c_int32), ("wide_lattice", C.c_int32), ("reserved", C.c_int32 * 3),
    ]


class JobC(C.Structure):            # qmc_job
    _fields_ = [
        ("sector", C.c_int32), ("shift_offset", C.c_int32), ("n", C.c_uint64), ("z", C.c_uint64 * MAXD),
        ("coef_re", C.c_double), ("coef_im", C.c_double),
    ]


class PieceC(C.Structure):          # qmc_piece
    _fields_ = [("job", C.c_int32), ("s0", C.c_int32), ("s1", C.c_int32), ("reserved", C.c_int32),
                ("k0", C.c_uint64), ("k1", C.c_uint64)]


class LaunchStats(C.Structure):     # qmc_launch_stats
    _fields_ = [("kernel_launches", C.c_int64), ("tiles", C.c_int64), ("evaluations", C.c_int64),
                ("eval_kernel_launches", C.c_int64)]


_lib = None


def lib():
    """Loads libqmc.so (fails loudly if it is missing) and declares the prototypes."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError("%s is missing: build it with `python -m paper_2305_19768_b200.build` "
                          "(there is no CPU fallback)" % LIB_PATH)
    L = C.CDLL(LIB_PATH)
    P, I32, U64, D = C.c_void_p, C.c_int32, C.c_uint64, C.c_double
    L.qmc_plan.restype = I32
    L.qmc_plan.argtypes = [P, I32, P, C.POINTER(P)]
    L.qmc_plan_orders.restype = I32
    L.qmc_plan_orders.argtypes = [P]
    L.qmc_plan_modules.restype = I32
    L.qmc_plan_modules.argtypes = [P]
    L.qmc_plan_module_source.restype = C.c_char_p
    L.qmc_plan_module_source.argtypes = [P, I32]
    L.qmc_plan_module_log.restype = C.c_char_p
    L.qmc_plan_module_log.argtypes = [P, I32]
    L.qmc_plan_sector_flops.restype = D
    L.qmc_plan_sector_flops.argtypes = [P, I32]
    L.qmc_plan_sector_ops.restype = D
    L.qmc_plan_sector_ops.argtypes = [P, I32]
    L.qmc_plan_sector_emitted_flops.restype = D
    L.qmc_plan_sector_emitted_flops.argtypes = [P, I32]
    L.qmc_plan_workspace_bytes.restype = C.c_size_t
    L.qmc_plan_workspace_bytes.argtypes = [P, I32, I32]
    L.qmc_plan_bind_workspace.restype = I32
    L.qmc_plan_bind_workspace.argtypes = [P, P, C.c_size_t]
    L.qmc_integrate_sectors.restype = I32
    L.qmc_integrate_sectors.argtypes = [P, P, I32, P, I32, I32, P, P, P, P, P]
    L.qmc_median_rule.restype = I32
    L.qmc_median_rule.argtypes = [P, I32, U64, P, I32, P, P, P, P, P]
    L.qmc_median_integrate_sectors.restype = I32
    L.qmc_median_integrate_sectors.argtypes = [P, P, I32, P, I32, P, P, I32, I32, P, P, P, P, P, P, P, P]
    L.qmc_debug_lattice_coords.restype = I32
    L.qmc_debug_lattice_coords.argtypes = [U64, P, I32, U64, U64, P, P]
    L.qmc_debug_eval_points.restype = I32
    L.qmc_debug_eval_points.argtypes = [P, I32, U64, P, P, P, I32, P, P]
    L.qmc_allocate_lattices.restype = I32
    L.qmc_allocate_lattices.argtypes = [P, P, P, I32, D, D, P]
    L.qmc_adaptive_scratch_bytes.restype = C.c_size_t
    L.qmc_adaptive_scratch_bytes.argtypes = [P, I32, P]
    L.qmc_adaptive_integrate.restype = I32
    L.qmc_adaptive_integrate.argtypes = [P, P, I32, P, P, P, C.c_size_t, P, P, P, P, P, P]
    L.qmc_debug_math_tables.restype = I32
    L.qmc_debug_math_tables.argtypes = [P, P, P]
    L.qmc_measure_fp64_peak.restype = I32
    L.qmc_measure_fp64_peak.argtypes = [D, C.POINTER(D), P]
    L.qmc_measure_fp64_peak_mixed.restype = I32
    L.qmc_measure_fp64_peak_mixed.argtypes = [D, C.POINTER(D), P]
    L.qmc_plan_last_stats.restype = I32
    L.qmc_plan_last_stats.argtypes = [P, C.POINTER(LaunchStats)]
    L.qmc_plan_last_eval_ms.restype = I32
    L.qmc_plan_last_eval_ms.argtypes = [P, C.POINTER(C.c_float)]
    L.qmc_integrate_pieces.restype = I32
    L.qmc_integrate_pieces.argtypes = [P, P, I32, P, I32, P, I32, I32, P, P, P]
    L.qmc_finalize_pieces.restype = I32
    L.qmc_finalize_pieces.argtypes = [P, P, I32, I32, P, I32, P, P, P, P]
    L.qmc_median_select_pieces.restype = I32
    L.qmc_median_select_pieces.argtypes = [P, P, I32, I32, P, I32, P, P, P, P]
    L.qmc_presample_scratch_bytes.restype = C.c_size_t
    L.qmc_presample_scratch_bytes.argtypes = [P, P]
    L.qmc_presample_lambda.restype = I32
    L.qmc_presample_lambda.argtypes = [P, U64, P, P, P, P, C.c_size_t, P, P]
    L.qmc_presample_static_max_bytes.restype = C.c_size_t
    L.qmc_presample_static_max_bytes.argtypes = []
    L.qmc_presample_lambda_static.restype = I32
    L.qmc_presample_lambda_static.argtypes = [P, U64, P, P, P, P, P]
    L.qmc_plan_last_job_clocks.restype = I32
    L.qmc_plan_last_job_clocks.argtypes = [P, P, I32]
    L.qmc_plan_slow_path_counts.restype = I32
    L.qmc_plan_slow_path_counts.argtypes = [P, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
    L.qmc_plan_destroy.restype = None
    L.qmc_plan_destroy.argtypes = [P]
    L.qmc_status_str.restype = C.c_char_p
    L.qmc_status_str.argtypes = [I32]
    L.qmc_last_error.restype = C.c_char_p
    L.qmc_last_error.argtypes = []
    _lib = L
    return L


def _status_str(status: int) -> str:
    return lib().qmc_status_str(int(status)).decode()


def _check(status: int):
    if status != QMC_OK:
        raise QmcError(status, lib().qmc_last_error().decode())


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _dptr(t):
    """Device pointer of a torch tensor (or None)."""
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream(stream) -> C.c_void_p:
    if stream is None:
        import torch
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))


def marshal_sector(s: W.Sector, keep: list) -> SectorDesc:
    """workloads.Sector -> qmc_sector_desc; the numpy arrays it points to are appended to keep."""
    if s.kind not in (W.KIND_UF, W.KIND_TOY):
        raise QmcError(QMC_ERR_UNSUPPORTED, "integrand kind %d is not part of the CUDA path" % s.kind)

    def k(arr, dtype):
        arr = np.ascontiguousarray(arr, dtype)
        keep.append(arr)
        return arr

    d = SectorDesc()
    d.kind, d.dim, d.transform, d.deformed = int(s.kind), int(s.dim), int(s.transform), int(s.deformed)
    d.first_order, d.n_orders = int(s.first_order), int(s.n_orders)
    for i in range(MAXD):
        d.a[i] = int(s.a[i])
    U_coef, F_coef = k(s.U_coef, np.float64), k(s.F_coef, np.float64)
    U_exp, F_exp = k(s.U_exp, np.uint8), k(s.F_exp, np.uint8)
    d.nU, d.nF = len(U_coef), (len(F_coef) if s.kind == W.KIND_UF else 0)
    d.p, d.q, d.lam, d.f_im = float(s.p), float(s.q), float(s.lam), float(s.f_im)
    d.U_coef, d.U_exp, d.F_coef, d.F_exp = _ptr(U_coef), _ptr(U_exp), _ptr(F_coef), _ptr(F_exp)
    d.logc = _ptr(k(s.logc, np.float64))
    return d


def marshal_jobs(jobs: Sequence[W.Job]):
    arr = (JobC * len(jobs))()
    for i, j in enumerate(jobs):
        arr[i].sector, arr[i].shift_offset, arr[i].n = int(j.sector), int(j.shift_offset), int(j.n)
        for k in range(MAXD):
            arr[i].z[k] = int(j.z[k]) if k < len(j.z) else 0
        arr[i].coef_re, arr[i].coef_im = float(np.real(j.coef)), float(np.imag(j.coef))
    return arr


class Plan:
    """Owner of a ``qmc_plan_t*`` and of the torch workspace tensor bound to it."""

    def __init__(self, handle: C.c_void_p, n_sectors: int):
        self.handle = handle
        self.n_sectors = n_sectors
        self.workspace = None
        self.J = lib().qmc_plan_orders(handle)

    # -- introspection (host only)
    def modules(self) -> int:
        return lib().qmc_plan_modules(self.handle)

    def module_source(self, i: int) -> str:
        return lib().qmc_plan_module_source(self.handle, i).decode()

    def module_log(self, i: int) -> str:
        return lib().qmc_plan_module_log(self.handle, i).decode()

    def sector_flops(self, i: int) -> float:
        return lib().qmc_plan_sector_flops(self.handle, i)

    def sector_ops(self, i: int) -> float:
        return lib().qmc_plan_sector_ops(self.handle, i)

    def sector_emitted_flops(self, i: int) -> float:
        return lib().qmc_plan_sector_emitted_flops(self.handle, i)

    def workspace_bytes(self, max_jobs: int, max_shift_rows: int) -> int:
        return lib().qmc_plan_workspace_bytes(self.handle, int(max_jobs), int(max_shift_rows))

    def bind_workspace(self, max_jobs: int, max_shift_rows: int, device="cuda:0"):
        """Allocates the workspace as a torch tensor (PyTorch is the only allocator) and binds it."""
        import torch
        nbytes = self.workspace_bytes(max_jobs, max_shift_rows)
        if nbytes == 0:
            raise QmcError(QMC_ERR_INVALID_ARG, "workspace_bytes returned 0")
        with torch.cuda.device(device):
            ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=device)
            off = (-ws.data_ptr()) % 256
            _check(lib().qmc_plan_bind_workspace(self.handle, C.c_void_p(ws.data_ptr() + off), nbytes))
        self.workspace = ws
        return self

    def last_stats(self) -> dict:
        st = LaunchStats()
        _check(lib().qmc_plan_last_stats(self.handle, C.byref(st)))
        return {f: getattr(st, f) for f, _ in LaunchStats._fields_}

    def last_eval_ms(self) -> float:
        ms = C.c_float()
        _check(lib().qmc_plan_last_eval_ms(self.handle, C.byref(ms)))
        return ms.value

    def last_job_clocks(self, n_rows: int) -> np.ndarray:
        """SM clock cycles spent in the tiles of each job of the last call (rows as in qmc.h); waits for the call."""
        out = np.zeros(int(n_rows), np.int64)
        _check(lib().qmc_plan_last_job_clocks(self.handle, _ptr(out), int(n_rows)))
        return out

    def slow_path_counts(self) -> dict:
        """Rare-path counters (waits for the plan's last call): evaluations re-done by the guarded evaluator, calls of
        the CUDA-library fallbacks."""
        a, b = C.c_int64(), C.c_int64()
        _check(lib().qmc_plan_slow_path_counts(self.handle, C.byref(a), C.byref(b)))
        return {"checked_evals": a.value, "slow_calls": b.value}

    def destroy(self):
        if self.handle is not None:
            lib().qmc_plan_destroy(self.handle)
            self.handle = None
            self.workspace = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def qmc_plan(sectors: Sequence[W.Sector], presample: int = 0, presample_opts: Optional[dict] = None, **opts) -> Plan:
    """qmc_plan: lowers the sector descriptions to generated CUDA and compiles it (no GPU needed).
    presample = N_PRE > 0 first runs qmc_presample_lambda on every deformed sector (on copies; needs a GPU) and
    plans with the selected deformation strengths: lambda is compiled into the sector's code."""
    if presample > 0:
        import copy
        sectors = [copy.deepcopy(s) for s in sectors]
        presample_sectors(sectors, n_pre=int(presample), **(presample_opts or {}))
    keep: list = []
    arr = (SectorDesc * max(1, len(sectors)))()
    for i, s in enumerate(sectors):
        arr[i] = marshal_sector(s, keep)
    o = PlanOpts()
    for key, val in opts.items():
        if not hasattr(o, key):
            raise TypeError("unknown plan option %r" % key)
        setattr(o, key, int(val))
    h = C.c_void_p()
    _check(lib().qmc_plan(C.cast(arr, C.c_void_p), len(sectors), C.cast(C.pointer(o), C.c_void_p), C.byref(h)))
    return Plan(h, len(sectors))


def _shifts8(shifts) -> np.ndarray:
    sh = np.ascontiguousarray(shifts, np.float64)
    if sh.ndim != 2 or sh.shape[1] != MAXD:
        raise ValueError("shifts must be rows x %d" % MAXD)
    return sh


def alloc_outputs(plan: Plan, n_jobs: int, m: int, K: int = 0, device="cuda:0", amplitude=True, diag=True) -> dict:
    """Caller-owned output tensors of one integrate / median call (zero-filled torch tensors)."""
    import torch
    J = plan.J
    f64 = dict(dtype=torch.float64, device=device)
    out = {
        "shift_sums": torch.zeros((n_jobs, m, J, 3), **f64),
        "job_results": torch.zeros((n_jobs, J, 4), **f64),
        "amplitude": torch.zeros((J, 4), **f64) if amplitude else None,
        "diag": torch.zeros((n_jobs, 2), dtype=torch.int64, device=device) if diag else None,
    }
    if K > 0:
        out["cand_est"] = torch.zeros((n_jobs, K, J, 2), **f64)
        out["median"] = torch.zeros((n_jobs, J, 2), **f64)
        out["selected"] = torch.zeros((n_jobs,), dtype=torch.int32, device=device)
    return out


def qmc_integrate_sectors(plan: Plan, jobs, shifts, m: int, out: dict, stream=None) -> None:
    """qmc_integrate_sectors: enqueue-only; results land in the tensors of ``out``."""
    jc = jobs if isinstance(jobs, C.Array) else marshal_jobs(jobs)
    sh = _shifts8(shifts)
    _check(lib().qmc_integrate_sectors(plan.handle, C.cast(jc, C.c_void_p), len(jc), _ptr(sh), sh.shape[0], int(m),
                                       _dptr(out["shift_sums"]), _dptr(out["job_results"]), _dptr(out.get("amplitude")),
                                       _dptr(out.get("diag")), _stream(stream)))


def qmc_median_integrate_sectors(plan: Plan, jobs, z_cand, shift0, shifts, m: int, out: dict, stream=None) -> None:
    """Batched median rule + m-shift integration on the selected vectors (config C2), enqueue-only."""
    jc = jobs if isinstance(jobs, C.Array) else marshal_jobs(jobs)
    zc = np.ascontiguousarray(z_cand, np.uint64)
    if zc.ndim != 3 or zc.shape[0] != len(jc) or zc.shape[2] != MAXD:
        raise ValueError("z_cand must be n_jobs x K x %d" % MAXD)
    s0 = _shifts8(shift0)
    if s0.shape[0] != len(jc):
        raise ValueError("shift0 must have one row per job")
    sh = _shifts8(shifts)
    _check(lib().qmc_median_integrate_sectors(
        plan.handle, C.cast(jc, C.c_void_p), len(jc), _ptr(zc), zc.shape[1], _ptr(s0), _ptr(sh), sh.shape[0], int(m),
        _dptr(out["cand_est"]), _dptr(out["median"]), _dptr(out["selected"]), _dptr(out["shift_sums"]),
        _dptr(out["job_results"]), _dptr(out.get("amplitude")), _dptr(out.get("diag")), _stream(stream)))


def marshal_pieces(pieces):
    """pieces: (job, s0, s1, k0, k1) tuples, sorted by job."""
    arr = (PieceC * max(1, len(pieces)))()
    for i, (job, s0, s1, k0, k1) in enumerate(pieces):
        arr[i].job, arr[i].s0, arr[i].s1, arr[i].k0, arr[i].k1 = int(job), int(s0), int(s1), int(k0), int(k1)
    return arr


def qmc_integrate_pieces(plan: Plan, jobs, pieces, shifts, m: int, d_partial, d_diag=None, stream=None) -> None:
    """qmc_integrate_pieces: this rank's pieces of a batch -> per-shift (hi, lo) partial sums, enqueue-only."""
    jc = jobs if isinstance(jobs, C.Array) else marshal_jobs(jobs)
    sh = _shifts8(shifts)
    pc = marshal_pieces(pieces)
    _check(lib().qmc_integrate_pieces(plan.handle, C.cast(jc, C.c_void_p), len(jc), C.cast(pc, C.c_void_p), len(pieces),
                                      _ptr(sh), sh.shape[0], int(m), _dptr(d_partial), _dptr(d_diag), _stream(stream)))


def qmc_finalize_pieces(plan: Plan, jobs, m: int, d_parts, n_parts: int, out: dict, stream=None) -> None:
    """qmc_finalize_pieces: the gathered partial sums of all ranks -> shift sums, mean / error, amplitude."""
    jc = jobs if isinstance(jobs, C.Array) else marshal_jobs(jobs)
    _check(lib().qmc_finalize_pieces(plan.handle, C.cast(jc, C.c_void_p), len(jc), int(m), _dptr(d_parts), int(n_parts),
                                     _dptr(out["shift_sums"]), _dptr(out["job_results"]), _dptr(out.get("amplitude")),
                                     _stream(stream)))


def qmc_median_select_pieces(plan: Plan, cand_jobs, K: int, d_parts, n_parts: int, out: dict, stream=None) -> None:
    """qmc_median_select_pieces: gathered candidate-stage parts (n_jobs K one-shift jobs) -> cand_est, median, selected."""
    jc = cand_jobs if isinstance(cand_jobs, C.Array) else marshal_jobs(cand_jobs)
    if len(jc) % int(K):
        raise ValueError("cand_jobs must hold n_jobs x K jobs")
    _check(lib().qmc_median_select_pieces(plan.handle, C.cast(jc, C.c_void_p), len(jc) // int(K), int(K), _dptr(d_parts),
                                          int(n_parts), _dptr(out["cand_est"]), _dptr(out["median"]), _dptr(out["selected"]),
                                          _stream(stream)))


def qmc_median_rule(plan: Plan, sector: int, n: int, z_cand, shift0, d_cand_est, d_median, d_selected, stream=None) -> None:
    """qmc_median_rule for one sector: K x J x 2 estimates, J x 2 medians, selected index (device tensors)."""
    zc = np.ascontiguousarray(z_cand, np.uint64)
    if zc.ndim != 2 or zc.shape[1] != MAXD:
        raise ValueError("z_cand must be K x %d" % MAXD)
    s0 = np.ascontiguousarray(shift0, np.float64).reshape(-1)
    if s0.shape[0] != MAXD:
        raise ValueError("shift0 must have %d entries" % MAXD)
    _check(lib().qmc_median_rule(plan.handle, int(sector), int(n), _ptr(zc), zc.shape[0], _ptr(s0), _dptr(d_cand_est),
                                 _dptr(d_median), _dptr(d_selected), _stream(stream)))


def qmc_debug_lattice_coords(n: int, z, dim: int, k0: int, count: int, d_out, stream=None) -> None:
    zz = np.zeros(MAXD, np.uint64)
    zz[:dim] = np.asarray(z, np.uint64)[:dim]
    _check(lib().qmc_debug_lattice_coords(int(n), _ptr(zz), int(dim), int(k0), int(count), _dptr(d_out), _stream(stream)))


def qmc_debug_eval_points(plan: Plan, sector: int, n: int, z, shift, ks, d_out, stream=None) -> None:
    zz = np.zeros(MAXD, np.uint64)
    z = np.asarray(z, np.uint64).ravel()
    zz[:len(z)] = z
    sh = np.zeros(MAXD, np.float64)
    shift = np.asarray(shift, np.float64).ravel()
    sh[:len(shift)] = shift
    kk = np.ascontiguousarray(ks, np.uint64)
    _check(lib().qmc_debug_eval_points(plan.handle, int(sector), int(n), _ptr(zz), _ptr(sh), _ptr(kk), len(kk),
                                       _dptr(d_out), _stream(stream)))


def debug_row_width(plan: Plan) -> int:
    """Doubles per point written by qmc_debug_eval_points: t[8], x[8], W, J x (re, im)."""
    return 2 * MAXD + 1 + 2 * plan.J


class PresampleOpts(C.Structure):
    _fields_ = [("lambda_max", C.c_double), ("decrease", C.c_double), ("lambda_min", C.c_double), ("min_abs_f", C.c_double)]


class PresampleInfo(C.Structure):
    _fields_ = [("lam", C.c_double), ("max_im_f", C.c_double), ("min_abs_f", C.c_double), ("steps", C.c_int32), ("ok", C.c_int32)]


def qmc_presample_lambda(sector: W.Sector, n_pre: int, z, shift, stream=None, device="cuda:0", **opts) -> dict:
    """qmc_presample_lambda: the largest admissible deformation strength of one deformed sector on n_pre presample
    points (every evaluation runs in the library's kernel); returns dict(lam, ok, steps, max_im_f, min_abs_f)."""
    import torch
    keep: list = []
    sd = marshal_sector(sector, keep)
    o = PresampleOpts()
    for key, val in opts.items():
        if not hasattr(o, key):
            raise TypeError("unknown presample option %r" % key)
        setattr(o, key, float(val))
    nbytes = lib().qmc_presample_scratch_bytes(C.byref(sd), C.byref(o))
    scratch = torch.empty(nbytes + 256, dtype=torch.uint8, device=device)
    off = (-scratch.data_ptr()) % 256
    zz = np.zeros(MAXD, np.uint64)
    zz[:sector.dim] = np.asarray(z, np.uint64).ravel()[:sector.dim]
    sh = np.zeros(MAXD, np.float64)
    sh[:sector.dim] = np.asarray(shift, np.float64).ravel()[:sector.dim]
    info = PresampleInfo()
    _check(lib().qmc_presample_lambda(C.byref(sd), int(n_pre), _ptr(zz), _ptr(sh), C.byref(o), C.c_void_p(scratch.data_ptr() + off),
                                      nbytes, C.byref(info), _stream(stream)))
    return {"lam": info.lam, "ok": bool(info.ok), "steps": info.steps, "max_im_f": info.max_im_f, "min_abs_f": info.min_abs_f}


def qmc_presample_lambda_static(sector: W.Sector, n_pre: int, z, shift, stream=None, **opts) -> dict:
    """qmc_presample_lambda_static: the same selection with the device scratch inside libqmc.so (96 KiB per GPU, F of
    at most 4096 monomials) -- the call allocates nothing, here or in the library; the stream's device must be current."""
    keep: list = []
    sd = marshal_sector(sector, keep)
    o = PresampleOpts()
    for key, val in opts.items():
        if not hasattr(o, key):
            raise TypeError("unknown presample option %r" % key)
        setattr(o, key, float(val))
    zz = np.zeros(MAXD, np.uint64)
    zz[:sector.dim] = np.asarray(z, np.uint64).ravel()[:sector.dim]
    sh = np.zeros(MAXD, np.float64)
    sh[:sector.dim] = np.asarray(shift, np.float64).ravel()[:sector.dim]
    info = PresampleInfo()
    _check(lib().qmc_presample_lambda_static(C.byref(sd), int(n_pre), _ptr(zz), _ptr(sh), C.byref(o), C.byref(info), _stream(stream)))
    return {"lam": info.lam, "ok": bool(info.ok), "steps": info.steps, "max_im_f": info.max_im_f, "min_abs_f": info.min_abs_f}


def presample_sectors(sectors: Sequence[W.Sector], n_pre: int = 100003, seed: int = 2305, device="cuda:0", **opts):
    """Sets s.lam of every deformed sector to its presampled value (in place; marshalling only: the lattice vector and
    the shift of the presample points are drawn here, the selection runs in qmc_presample_lambda).  Returns the infos.
    Call before qmc_plan: lambda is compiled into the sector's code."""
    rng = np.random.Generator(np.random.PCG64(seed))
    infos = []
    for s in sectors:
        if not s.deformed:
            infos.append(None)
            continue
        z = W.draw_z(rng, n_pre, s.dim)
        shift = W.draw_shifts(rng, 1, s.dim)[0]
        r = qmc_presample_lambda(s, n_pre, z, shift, device=device, **opts)
        s.lam = r["lam"]
        infos.append(r)
    return infos


class AdaptiveOpts(C.Structure):
    _fields_ = [("epsrel", C.c_double), ("epsabs", C.c_double), ("alpha", C.c_double), ("growth_max", C.c_double),
                ("safety", C.c_double), ("n_min", C.c_uint64), ("n_max", C.c_uint64), ("seed", C.c_uint64),
                ("max_rounds", C.c_int32), ("m", C.c_int32), ("K", C.c_int32), ("measure_tau", C.c_int32)]


class AdaptiveInfo(C.Structure):
    _fields_ = [("rounds", C.c_int32), ("converged", C.c_int32), ("evaluations", C.c_int64)]


def qmc_allocate_lattices(w, tau, c_abs2, alpha: float, V: float) -> np.ndarray:
    """Eq. (6) of the paper through the library (host arithmetic; needs no GPU)."""
    w, tau, c2 = (np.ascontiguousarray(a, np.float64) for a in (w, tau, c_abs2))
    out = np.zeros(len(w))
    _check(lib().qmc_allocate_lattices(_ptr(w), _ptr(tau), _ptr(c2), len(w), float(alpha), float(V), _ptr(out)))
    return out


def qmc_adaptive_integrate(plan: Plan, jobs, tau=None, stream=None, device="cuda:0", **opts) -> dict:
    """qmc_adaptive_integrate: allocates the workspace and the device scratch as torch tensors, marshals the
    arguments and returns the host outputs.  Every round's evaluation runs in the library's kernels."""
    import torch
    o = AdaptiveOpts()
    for key, val in opts.items():
        if not hasattr(o, key):
            raise TypeError("unknown adaptive option %r" % key)
        setattr(o, key, val)
    jc = jobs if isinstance(jobs, C.Array) else marshal_jobs(jobs)
    nj = len(jc)
    m, K = (o.m or 32), (o.K or 11)
    plan.bind_workspace(nj * (K + 1), nj * (m + 1), device=device)
    nbytes = lib().qmc_adaptive_scratch_bytes(plan.handle, nj, C.byref(o))
    scratch = torch.empty(nbytes + 256, dtype=torch.uint8, device=device)
    off = (-scratch.data_ptr()) % 256
    J = plan.J
    res, amp = np.zeros((nj, J, 4)), np.zeros((J, 4))
    n_final, z_final = np.zeros(nj, np.uint64), np.zeros((nj, W.QMC_MAX_DIM), np.uint64)
    info = AdaptiveInfo()
    tau_a = None if tau is None else np.ascontiguousarray(tau, np.float64)
    _check(lib().qmc_adaptive_integrate(plan.handle, C.cast(jc, C.c_void_p), nj, None if tau_a is None else _ptr(tau_a),
                                        C.byref(o), C.c_void_p(scratch.data_ptr() + off), nbytes, _ptr(res), _ptr(amp),
                                        _ptr(n_final), _ptr(z_final), C.byref(info), _stream(stream)))
    return {"job_results": res, "amplitude": amp, "n_final": n_final, "z_final": z_final, "rounds": info.rounds,
            "converged": info.converged, "evaluations": info.evaluations}


def qmc_debug_math_tables():
    """The lookup tables of the library's own log / exp / sincos / atan2 (host arrays; needs no GPU)."""
    lt, et, tt = np.zeros(2050), np.zeros(256), np.zeros(512)
    _check(lib().qmc_debug_math_tables(_ptr(lt), _ptr(et), _ptr(tt)))
    return lt, et, tt


def qmc_measure_fp64_peak_mixed(millis: float = 200.0, stream=None) -> float:
    out = C.c_double()
    _check(lib().qmc_measure_fp64_peak_mixed(float(millis), C.byref(out), _stream(stream)))
    return out.value


def qmc_measure_fp64_peak(millis: float = 200.0, stream=None) -> float:
    out = C.c_double()
    _check(lib().qmc_measure_fp64_peak(float(millis), C.byref(out), _stream(stream)))
    return out.value
