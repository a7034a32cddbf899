"""TEST INFRASTRUCTURE, NOT THE PRODUCT -- oracle of the deformation-parameter presampling.

The paper says only that `number_of_presamples` is "the number of samples used for the initial contour deformation
parameter selection" and that the deformation must keep the sign of Im F (the check counted in
diag[1], A5).  Reading R-pre, step by step:

  1. presample points: the n_pre points x_k of ONE shifted rank-1 lattice (A1-A3 with the sector's own transform);
     points of weight 0 are skipped (they do not enter any sum);
  2. candidates: lambda_0 = lambda_max, lambda_{j+1} = lambda_j * decrease (one multiplication per step), as long as
     lambda_j >= lambda_min;
  3. a candidate is ADMISSIBLE if at every presample point Im F(z(x_k; lambda_j)) < 0 (the sign check of A5, with the
     sector's f_im) and |F(z(x_k; lambda_j))| >= min_abs_f (distance of the contour from the zeros of F; 0 = off);
  4. the result is the first (largest) admissible candidate (ok = True).  If none is admissible: among the candidates
     that pass the sign check at every point, the one whose contour stays farthest from the zeros of F (largest
     min_k |F|; the larger lambda on a tie) is returned with ok = False; if no candidate passes the sign check,
     lambda_min is returned with ok = False.

Plain Python over the oracle's own A1-A3 and orc_deformed_f; shares no code with the CUDA library.
"""
from __future__ import annotations

import numpy as np


def candidates(lambda_max=1.0, decrease=0.9, lambda_min=1e-5):
    out, lam = [], float(lambda_max)
    while lam >= lambda_min:
        out.append(lam)
        lam = lam * decrease
    return out


def presample_lambda(sector, n_pre, z, shift, lambda_max=1.0, decrease=0.9, lambda_min=1e-5, min_abs_f=0.0):
    """Returns dict(lam, ok, steps, max_im_f, min_abs_f) -- the last two are taken over the presample points at the
    returned lambda."""
    from oracle import oracle as O
    sec = O.OracleSector(sector)
    xs = []
    for k in range(int(n_pre)):
        _t, x, W, _wg, _sf = O.eval_point(sec, int(n_pre), z, shift, k)
        if W != 0.0:
            xs.append(np.array(x))
    cands = candidates(lambda_max, decrease, lambda_min)
    best = None                                     # fallback: (min |F|, lambda, index, max Im F) of the best sign-admissible candidate
    for j, lam in enumerate(cands):
        worst_im, least_abs, sign_ok = -np.inf, np.inf, True
        for x in xs:
            f = O.deformed_f(sec, x, lam)
            worst_im = max(worst_im, f.imag)
            least_abs = min(least_abs, abs(f))
            if not (f.imag < 0.0):
                sign_ok = False
                break
        if not sign_ok:
            continue
        if least_abs >= min_abs_f:
            return {"lam": lam, "ok": True, "steps": j, "max_im_f": worst_im, "min_abs_f": least_abs}
        if best is None or least_abs > best[0]:
            best = (least_abs, lam, j, worst_im)
    if best is not None:
        return {"lam": best[1], "ok": False, "steps": best[2], "max_im_f": best[3], "min_abs_f": best[0]}
    return {"lam": float(lambda_min), "ok": False, "steps": len(cands), "max_im_f": float("nan"), "min_abs_f": float("nan")}
