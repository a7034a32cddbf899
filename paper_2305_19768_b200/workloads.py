"""Seeded synthetic input generators for the QMC hot path (configs C0..C4 of BASELINE.json).

This module is INPUT ONLY: it draws sector descriptions (polynomial exponents and
coefficients, powers, log-polynomial coefficients), lattice sizes, generating vectors
and shifts from a seeded numpy generator.  It contains none of the method's arithmetic
(no lattice rule, no transform, no integrand evaluation, no reduction) and imports
neither the CUDA binding nor anything under ``oracle/``; both sides read the same
arrays from here.

The recipe follows SURVEY.md section 8(d) ("Concrete inputs") and the readings
Q8, Q11, Q12, Q13, Q17, Q18 of section 8(c).2; it is restated in DESIGN.md section 4.
The paper's own benchmark integrals need pySecDec's symbolic
stage and are not available; these synthetic sectors stand in for them.
"""
from __future__ import annotations

import itertools
import math
from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np

QMC_MAX_DIM = 8
MASTER_SEED = 2305

KIND_UF = 0      # x^a U^p F^q L(log U, log F)
KIND_TOY = 1     # prod_i (1 + c_i (x_i - 1/2) + d_i x_i^2)
KIND_TRIG = 2    # c0 + sum_h c_h cos(2 pi h.x + phi_h)   (oracle pin P5 only)

TRANSFORM_NONE = 0
TRANSFORM_KOROBOV3 = 1
TRANSFORM_BAKER = 2


# ----------------------------------------------------------------------------- primes
def _is_prime(n: int) -> bool:
    """Deterministic Miller-Rabin for n < 3.3e24 (first 13 prime bases)."""
    if n < 2:
        return False
    small = (2, 3, 5, 7, 11, 13, 17, 19, 23, 29, 31, 37, 41)
    for p in small:
        if n % p == 0:
            return n == p
    d, s = n - 1, 0
    while d % 2 == 0:
        d //= 2
        s += 1
    for a in small:
        x = pow(a, d, n)
        if x in (1, n - 1):
            continue
        for _ in range(s - 1):
            x = x * x % n
            if x == n - 1:
                break
        else:
            return False
    return True


def nearest_prime(x: float) -> int:
    """Prime nearest to the real number x; ties go to the lower prime."""
    c = int(round(x))
    for delta in range(0, 10_000):
        lo, hi = c - delta, c + delta
        lo_ok = lo >= 2 and _is_prime(lo)
        hi_ok = _is_prime(hi)
        if lo_ok and hi_ok:
            return lo if abs(x - lo) <= abs(hi - x) else hi
        if lo_ok:
            return lo
        if hi_ok:
            return hi
    raise ValueError("no prime found near %r" % (x,))


# ----------------------------------------------------------------------------- data
@dataclass
class Sector:
    dim: int
    kind: int = KIND_UF
    transform: int = TRANSFORM_KOROBOV3
    deformed: int = 0
    first_order: int = 0
    n_orders: int = 1
    a: np.ndarray = field(default_factory=lambda: np.zeros(QMC_MAX_DIM, np.int32))
    p: float = 0.0
    q: float = 0.0
    U_coef: np.ndarray = field(default_factory=lambda: np.ones(1))
    U_exp: np.ndarray = field(default_factory=lambda: np.zeros((1, 1), np.uint8))
    F_coef: np.ndarray = field(default_factory=lambda: np.ones(1))
    F_exp: np.ndarray = field(default_factory=lambda: np.zeros((1, 1), np.uint8))
    lam: float = 0.0
    f_im: float = 0.0
    logc: np.ndarray = field(default_factory=lambda: np.ones(1))
    # KIND_TRIG only: integer frequencies (nh x dim), amplitudes, phases; c0 in logc[0]
    trig_h: Optional[np.ndarray] = None
    trig_amp: Optional[np.ndarray] = None
    trig_phase: Optional[np.ndarray] = None

    def n_logc(self) -> int:
        return sum((j + 1) * (j + 2) // 2 for j in range(self.first_order, self.first_order + self.n_orders))


@dataclass
class Job:
    sector: int
    n: int
    z: np.ndarray                # uint64[QMC_MAX_DIM]
    shift_offset: int = 0        # first row of this job's m shifts in Workload.shifts
    coef: complex = 1.0 + 0.0j   # amplitude weight C_i


@dataclass
class Workload:
    name: str
    sectors: List[Sector]
    jobs: List[Job]
    shifts: np.ndarray           # float64[rows, QMC_MAX_DIM]
    m: int
    # median rule inputs (C2): per job K candidate vectors and one shared shift
    z_cand: Optional[np.ndarray] = None   # uint64[n_jobs, K, QMC_MAX_DIM]
    shift0: Optional[np.ndarray] = None   # float64[n_jobs, QMC_MAX_DIM]

    def evaluations(self) -> int:
        K = 0 if self.z_cand is None else self.z_cand.shape[1]
        return sum(j.n * (self.m + K) for j in self.jobs)

    def subset(self, idx) -> "Workload":
        """The jobs `idx` of this workload as a workload of their own (one rank's shard of a batch): sectors and
        shift rows are kept whole, so sector indices and shift offsets stay valid."""
        idx = list(idx)
        return Workload(self.name, self.sectors, [self.jobs[i] for i in idx], self.shifts, self.m,
                        None if self.z_cand is None else self.z_cand[idx],
                        None if self.shift0 is None else self.shift0[idx])


# ----------------------------------------------------------------------------- draws
def draw_shifts(rng: np.random.Generator, rows: int, dim: int) -> np.ndarray:
    """Delta = (u64 >> 11) * 2^-53, zeros redrawn; unused columns are 0."""
    out = np.zeros((rows, QMC_MAX_DIM), np.float64)
    for r in range(rows):
        for i in range(dim):
            v = 0
            while v == 0:
                v = int(rng.integers(0, 2**64, dtype=np.uint64)) >> 11
            out[r, i] = v * 2.0**-53
    return out


def draw_z(rng: np.random.Generator, n: int, dim: int) -> np.ndarray:
    """Each component uniform on the units mod n (Eq. 7)."""
    z = np.zeros(QMC_MAX_DIM, np.uint64)
    if n == 1:                      # the only residue mod 1 is 0 (degenerate one-point lattice)
        return z
    for i in range(dim):
        while True:
            c = int(rng.integers(1, n))
            if math.gcd(c, n) == 1:
                z[i] = c
                break
    return z


def _exponent_vectors(dim: int, deg_lo: int, deg_hi: int) -> np.ndarray:
    rows = []
    for deg in range(deg_lo, deg_hi + 1):
        for combo in itertools.combinations_with_replacement(range(dim), deg):
            e = [0] * dim
            for i in combo:
                e[i] += 1
            rows.append(e)
    return np.array(rows, np.uint8)


def draw_polynomial(rng, dim, n_mono, deg_lo, deg_hi, c_lo, c_hi, const_term=1.0):
    """1 + n_mono distinct monomials of total degree deg_lo..deg_hi (the
    constant term is the first row, not counted in n_mono; const_term=None drops it)."""
    pool = _exponent_vectors(dim, deg_lo, deg_hi)
    pick = rng.choice(len(pool), size=n_mono, replace=False)
    exps = pool[np.sort(pick)]
    coef = rng.uniform(c_lo, c_hi, size=n_mono)
    if const_term is not None:
        exps = np.vstack([np.zeros((1, dim), np.uint8), exps])
        coef = np.concatenate([[const_term], coef])
    return np.ascontiguousarray(coef, np.float64), np.ascontiguousarray(exps, np.uint8)


def n_monomials(dim: int):
    """nU(d) = 3(d-2), nF(d) = (d-2)(d+1)  (d=4 -> 6,10; d=6 -> 12,28)."""
    return max(1, 3 * (dim - 2)), max(1, (dim - 2) * (dim + 1))


def draw_euclid_sector(rng, dim, first_order=1, n_orders=1, const_term=1.0) -> Sector:
    """BASELINE.json config 1 recipe: x^a U^p F^q (c0 + c1 log F + c2 log U)."""
    nU, nF = n_monomials(dim)
    a = np.zeros(QMC_MAX_DIM, np.int32)
    a[:dim] = rng.integers(0, 2, size=dim)
    U_coef, U_exp = draw_polynomial(rng, dim, nU, 1, 2, 0.1, 1.0, const_term)
    F_coef, F_exp = draw_polynomial(rng, dim, nF, 2, 3, 0.1, 1.0, const_term)
    p, q = rng.uniform(-3.0, -0.5, size=2)
    s = Sector(dim=dim, kind=KIND_UF, transform=TRANSFORM_KOROBOV3, deformed=0,
               first_order=first_order, n_orders=n_orders, a=a, p=float(p), q=float(q),
               U_coef=U_coef, U_exp=U_exp, F_coef=F_coef, F_exp=F_exp)
    s.logc = _draw_logc(rng, first_order, n_orders)
    return s


def _draw_logc(rng, first_order, n_orders):
    """Order j: (j+1)(j+2)/2 coefficients of lU^alpha lF^beta, alpha+beta<=j, ordered by
    (alpha+beta, beta).  For j=1 the draw (c0, c1, c2) is stored as [c0, c2, c1] so that
    c1 multiplies log F and c2 multiplies log U as BASELINE.json config 1 writes it."""
    out = []
    for j in range(first_order, first_order + n_orders):
        c = rng.standard_normal((j + 1) * (j + 2) // 2)
        if j == 1:
            c = c[[0, 2, 1]]
        out.append(c)
    return np.ascontiguousarray(np.concatenate(out), np.float64)


def draw_physical_sector(rng, dim, lam=0.5, f_im=-1e-12) -> Sector:
    """BASELINE.json config 3 recipe: F has mixed-sign coefficients,
    contour deformation with lambda, orders eps^-2..eps^0 (J=3), baker transform."""
    nU, nF = n_monomials(dim)
    a = np.zeros(QMC_MAX_DIM, np.int32)
    a[:dim] = rng.integers(0, 2, size=dim)
    U_coef, U_exp = draw_polynomial(rng, dim, nU, 1, 2, 0.1, 1.0, 1.0)
    F_coef, F_exp = draw_polynomial(rng, dim, nF, 2, 3, -1.0, 1.0, 1.0)
    p, q = rng.uniform(-3.0, -0.5, size=2)
    s = Sector(dim=dim, kind=KIND_UF, transform=TRANSFORM_BAKER, deformed=1,
               first_order=0, n_orders=3, a=a, p=float(p), q=float(q),
               U_coef=U_coef, U_exp=U_exp, F_coef=F_coef, F_exp=F_exp,
               lam=float(lam), f_im=float(f_im))
    s.logc = _draw_logc(rng, 0, 3)
    return s


# ----------------------------------------------------------------------------- configs
def _seed(config_id: int) -> int:
    return MASTER_SEED * 100 + config_id


def config_toy(n: int = 65521, m: int = 32, dim: int = 2, seed: Optional[int] = None) -> Workload:
    """C0: dim=2 separable integrand, exact integral prod_i (1 + d_i/3)."""
    rng = np.random.Generator(np.random.PCG64(_seed(0) if seed is None else seed))
    c = rng.uniform(-1.0, 1.0, size=dim)
    d = rng.uniform(-1.0, 1.0, size=dim)
    s = Sector(dim=dim, kind=KIND_TOY, transform=TRANSFORM_KOROBOV3,
               U_coef=np.ascontiguousarray(np.concatenate([c, d])),
               U_exp=np.zeros((2 * dim, dim), np.uint8))
    z = draw_z(rng, n, dim)
    shifts = draw_shifts(rng, m, dim)
    return Workload("C0-toy", [s], [Job(0, n, z, 0)], shifts, m)


def toy_exact(s: Sector) -> float:
    """Closed form of the C0 integral (input-side bookkeeping: prod_i (1 + d_i/3))."""
    d = s.U_coef[s.dim:2 * s.dim]
    return float(np.prod(1.0 + d / 3.0))


def config_euclid(n_sectors: int = 8, dim: int = 4, n: Optional[int] = None, m: int = 32,
                  seed: Optional[int] = None, const_term=1.0) -> Workload:
    """C1: 8 Euclidean sectors of dim 4 at n = prime nearest 2^20 (1 048 573)."""
    rng = np.random.Generator(np.random.PCG64(_seed(1) if seed is None else seed))
    if n is None:
        n = nearest_prime(2**20)
    sectors = [draw_euclid_sector(rng, dim, const_term=const_term) for _ in range(n_sectors)]
    jobs, rows = [], []
    for i in range(n_sectors):
        z = draw_z(rng, n, dim)
        jobs.append(Job(i, n, z, i * m))
        rows.append(draw_shifts(rng, m, dim))
    return Workload("C1-euclid", sectors, jobs, np.vstack(rows), m)


def config_median(n_sectors: int = 64, dim: int = 6, n: int = 1_000_003, K: int = 11, m: int = 32,
                  seed: Optional[int] = None) -> Workload:
    """C2: 64 Euclidean sectors of dim 6; K=11 candidate z per sector with one shared
    shift, then m shifts on the selected candidate."""
    rng = np.random.Generator(np.random.PCG64(_seed(2) if seed is None else seed))
    sectors = [draw_euclid_sector(rng, dim) for _ in range(n_sectors)]
    jobs, rows = [], []
    z_cand = np.zeros((n_sectors, K, QMC_MAX_DIM), np.uint64)
    shift0 = np.zeros((n_sectors, QMC_MAX_DIM), np.float64)
    for i in range(n_sectors):
        for k in range(K):
            z_cand[i, k] = draw_z(rng, n, dim)
        shift0[i] = draw_shifts(rng, 1, dim)[0]
        # Job.z is a placeholder (candidate 0) until the median rule selects j*
        jobs.append(Job(i, n, z_cand[i, 0].copy(), i * m))
        rows.append(draw_shifts(rng, m, dim))
    return Workload("C2-median", sectors, jobs, np.vstack(rows), m, z_cand=z_cand, shift0=shift0)


def config_physical(n_sectors: int = 32, dim: int = 5, n: int = 9_999_991, m: int = 32,
                    lam: float = 0.5, seed: Optional[int] = None) -> Workload:
    """C3: 32 contour-deformed sectors of dim 5, J=3 orders, baker transform."""
    rng = np.random.Generator(np.random.PCG64(_seed(3) if seed is None else seed))
    sectors = [draw_physical_sector(rng, dim, lam=lam) for _ in range(n_sectors)]
    jobs, rows = [], []
    for i in range(n_sectors):
        z = draw_z(rng, n, dim)
        jobs.append(Job(i, n, z, i * m))
        rows.append(draw_shifts(rng, m, dim))
    return Workload("C3-physical", sectors, jobs, np.vstack(rows), m)


def config_batch(n_sectors: int = 600, scale: float = 1.0, m: int = 32,
                 log10_n=(6.0, 9.0), seed: Optional[int] = None) -> Workload:
    """C4: 600 sectors of dims 3..8, 40 % deformed, complex weights, log-uniform n.
    ``scale`` divides every drawn n (1/28 gives the ~1e11 'C4-lite')."""
    rng = np.random.Generator(np.random.PCG64(_seed(4) if seed is None else seed))
    sectors, jobs, rows = [], [], []
    for i in range(n_sectors):
        dim = int(rng.integers(3, 9))
        deformed = bool(rng.uniform() < 0.4)
        s = draw_physical_sector(rng, dim) if deformed else draw_euclid_sector(rng, dim)
        n = nearest_prime(max(11.0, 10.0 ** rng.uniform(*log10_n) * scale))
        coef = complex(rng.standard_normal(), rng.standard_normal())
        z = draw_z(rng, n, dim)
        sectors.append(s)
        jobs.append(Job(i, n, z, i * m, coef))
        rows.append(draw_shifts(rng, m, dim))
    return Workload("C4-batch", sectors, jobs, np.vstack(rows), m)
