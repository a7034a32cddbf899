"""ctypes access to the CPU oracle (oracle/qmc_oracle.cpp) -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this module.  It builds the plain C++ oracle with g++ (``-O2 -std=c++17
-ffp-contract=off``) into ``oracle/libqmc_oracle.so`` on first use and marshals the seeded
inputs of ``paper_2305_19768_b200.workloads`` into the oracle's own ``orc_sector`` layout.
It contains no arithmetic of the method; every number comes out of qmc_oracle.cpp.
It does not import the CUDA binding and shares nothing with csrc/.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "qmc_oracle.cpp")
_LIB = os.path.join(_HERE, "libqmc_oracle.so")
MAXD = 8
_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle if the .so is missing or older than its source."""
    with _lock:
        stale = force or (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
        if stale:
            tmp = _LIB + ".tmp.%d" % os.getpid()
            subprocess.check_call(["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-shared", "-fPIC",
                                   "-o", tmp, _SRC])
            os.replace(tmp, _LIB)
    return _LIB


class _OrcSector(C.Structure):
    _fields_ = [
        ("kind", C.c_int32), ("dim", C.c_int32), ("transform", C.c_int32), ("deformed", C.c_int32),
        ("first_order", C.c_int32), ("n_orders", C.c_int32),
        ("a", C.c_int32 * MAXD),
        ("nU", C.c_int32), ("nF", C.c_int32),
        ("p", C.c_double), ("q", C.c_double), ("lam", C.c_double), ("f_im", C.c_double),
        ("U_coef", C.c_void_p), ("U_exp", C.c_void_p),
        ("F_coef", C.c_void_p), ("F_exp", C.c_void_p),
        ("logc", C.c_void_p),
        ("n_trig", C.c_int32), ("pad_", C.c_int32),
        ("trig_h", C.c_void_p), ("trig_amp", C.c_void_p), ("trig_phase", C.c_void_p),
    ]


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        P = C.c_void_p
        L.orc_n_orders.restype = C.c_int32
        L.orc_n_orders.argtypes = [P]
        L.orc_lattice_coords.restype = None
        L.orc_lattice_coords.argtypes = [C.c_uint64, P, C.c_int32, C.c_uint64, C.c_uint64, P]
        L.orc_eval_point.restype = None
        L.orc_eval_point.argtypes = [P, C.c_uint64, P, P, C.c_uint64, P, P, P, P, P]
        L.orc_integrand.restype = None
        L.orc_integrand.argtypes = [P, P, P, P]
        L.orc_deformation.restype = None
        L.orc_deformation.argtypes = [P, P, P, P]
        L.orc_deformed_f.restype = None
        L.orc_deformed_f.argtypes = [P, P, C.c_double, P]
        L.orc_shift_sums.restype = None
        L.orc_shift_sums.argtypes = [P, C.c_uint64, P, P, C.c_int32, C.c_uint64, C.c_uint64, P, P]
        L.orc_mean_err.restype = None
        L.orc_mean_err.argtypes = [P, C.c_int32, C.c_int32, C.c_uint64, P]
        L.orc_integrate.restype = None
        L.orc_integrate.argtypes = [P, C.c_uint64, P, P, C.c_int32, P, P, P]
        L.orc_median_rule.restype = None
        L.orc_median_rule.argtypes = [P, C.c_uint64, P, C.c_int32, P, P, P, P]
        L.orc_amplitude.restype = None
        L.orc_amplitude.argtypes = [P, P, C.c_int32, C.c_int32, P]
        _lib = L
    return _lib


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


class OracleSector:
    """Holds an ``orc_sector`` plus the numpy arrays its pointers refer to."""

    def __init__(self, s):
        d = int(s.dim)
        self._keep = []

        def keep(arr, dtype):
            arr = np.ascontiguousarray(arr, dtype)
            self._keep.append(arr)
            return arr

        o = _OrcSector()
        o.kind, o.dim, o.transform, o.deformed = int(s.kind), d, int(s.transform), int(s.deformed)
        o.first_order, o.n_orders = int(s.first_order), int(s.n_orders)
        for i in range(MAXD):
            o.a[i] = int(s.a[i])
        U_coef, F_coef = keep(s.U_coef, np.float64), keep(s.F_coef, np.float64)
        U_exp, F_exp = keep(s.U_exp, np.uint8), keep(s.F_exp, np.uint8)
        o.nU, o.nF = len(U_coef), len(F_coef)
        if s.kind == 0:
            assert U_exp.shape == (o.nU, d) and F_exp.shape == (o.nF, d)
        o.p, o.q, o.lam, o.f_im = float(s.p), float(s.q), float(s.lam), float(s.f_im)
        o.U_coef, o.U_exp, o.F_coef, o.F_exp = _ptr(U_coef), _ptr(U_exp), _ptr(F_coef), _ptr(F_exp)
        o.logc = _ptr(keep(s.logc, np.float64))
        if s.trig_h is not None:
            h = keep(s.trig_h, np.int32)
            o.n_trig = h.shape[0]
            o.trig_h, o.trig_amp, o.trig_phase = _ptr(h), _ptr(keep(s.trig_amp, np.float64)), _ptr(keep(s.trig_phase, np.float64))
        self.c = o
        self.dim = d
        self.J = lib().orc_n_orders(C.byref(o))

    @property
    def ref(self):
        return C.byref(self.c)


def _z8(z):
    out = np.zeros(MAXD, np.uint64)
    z = np.asarray(z, np.uint64).ravel()
    out[:len(z)] = z
    return out


def _shifts8(shifts):
    sh = np.atleast_2d(np.asarray(shifts, np.float64))
    out = np.zeros((sh.shape[0], MAXD), np.float64)
    out[:, :sh.shape[1]] = sh
    return out


def lattice_coords(n, z, dim, k0, count):
    """A1: r[k - k0, i] = (k * z_i) mod n for k in [k0, k0 + count)."""
    zz = _z8(z)
    out = np.zeros((count, dim), np.uint64)
    lib().orc_lattice_coords(int(n), _ptr(zz), int(dim), int(k0), int(count), _ptr(out))
    return out


def eval_point(sec: OracleSector, n, z, delta, k):
    """A1-A5 at lattice index k: returns (t[dim], x[dim], W, wg[J] complex, sign_fail)."""
    zz, dl = _z8(z), _shifts8(delta)[0]
    t, x = np.zeros(MAXD), np.zeros(MAXD)
    W = C.c_double()
    wg = np.zeros(2 * sec.J)
    sf = C.c_int32()
    lib().orc_eval_point(sec.ref, int(n), _ptr(zz), _ptr(dl), int(k), _ptr(t), _ptr(x), C.byref(W), _ptr(wg), C.byref(sf))
    return t[:sec.dim], x[:sec.dim], W.value, wg[0::2] + 1j * wg[1::2], sf.value


def integrand(sec: OracleSector, x):
    """A4 / A4' / A5 at a given point x (no transform, no weight): g[J] complex, sign_fail."""
    xx = np.zeros(MAXD)
    xx[:sec.dim] = x
    g = np.zeros(2 * sec.J)
    sf = C.c_int32()
    lib().orc_integrand(sec.ref, _ptr(xx), _ptr(g), C.byref(sf))
    return g[0::2] + 1j * g[1::2], sf.value


def deformation(sec: OracleSector, x):
    """A5: the deformed point z(x) (complex[dim]) and Jac = det M."""
    xx = np.zeros(MAXD)
    xx[:sec.dim] = x
    zo, jac = np.zeros(2 * MAXD), np.zeros(2)
    lib().orc_deformation(sec.ref, _ptr(xx), _ptr(zo), _ptr(jac))
    return (zo[0::2] + 1j * zo[1::2])[:sec.dim], complex(jac[0], jac[1])


def deformed_f(sec: OracleSector, x, lam) -> complex:
    """F(z(x; lam)) + i f_im for a given deformation strength (A5's sign-check quantity)."""
    xx = np.zeros(MAXD)
    xx[:sec.dim] = x
    f = np.zeros(2)
    lib().orc_deformed_f(sec.ref, _ptr(xx), float(lam), _ptr(f))
    return complex(f[0], f[1])


def shift_sums(sec: OracleSector, n, z, shifts, k0=0, k1=None):
    """A1-A6: sums[m, J, 3] = (Re S, Im S, sum |W g|) over k in [k0, k1); diag[2]."""
    zz, sh = _z8(z), _shifts8(shifts)
    m = sh.shape[0]
    sums = np.zeros((m, sec.J, 3))
    diag = np.zeros(2, np.int64)
    lib().orc_shift_sums(sec.ref, int(n), _ptr(zz), _ptr(sh), m, int(k0), int(n if k1 is None else k1), _ptr(sums), _ptr(diag))
    return sums, diag


def mean_err(sums, n):
    """A7: result[J, 4] = (mean_re, mean_im, err_re, err_im)."""
    sums = np.ascontiguousarray(sums, np.float64)
    m, J = sums.shape[0], sums.shape[1]
    res = np.zeros((J, 4))
    lib().orc_mean_err(_ptr(sums), m, J, int(n), _ptr(res))
    return res


def integrate(sec: OracleSector, n, z, shifts):
    """A1-A7 for one job: (sums[m, J, 3], result[J, 4], diag[2])."""
    sums, diag = shift_sums(sec, n, z, shifts)
    return sums, mean_err(sums, n), diag


def median_rule(sec: OracleSector, n, z_cand, shift0):
    """A8: (cand_est[K, J] complex, median[J] complex, selected index)."""
    zc = np.ascontiguousarray(z_cand, np.uint64)
    K = zc.shape[0]
    assert zc.shape[1] == MAXD
    s0 = _shifts8(shift0)[0]
    est, med = np.zeros((K, sec.J, 2)), np.zeros((sec.J, 2))
    sel = C.c_int32()
    lib().orc_median_rule(sec.ref, int(n), _ptr(zc), K, _ptr(s0), _ptr(est), _ptr(med), C.byref(sel))
    return est[..., 0] + 1j * est[..., 1], med[:, 0] + 1j * med[:, 1], sel.value


def amplitude(results, coefs):
    """A9: results[n_jobs, J, 4], coefs[n_jobs] complex -> amp[J, 4]."""
    results = np.ascontiguousarray(results, np.float64)
    nj, J = results.shape[0], results.shape[1]
    cf = np.zeros((nj, 2))
    cf[:, 0], cf[:, 1] = np.real(coefs), np.imag(coefs)
    amp = np.zeros((J, 4))
    lib().orc_amplitude(_ptr(results), _ptr(cf), nj, J, _ptr(amp))
    return amp
