"""Error metrics of the parity bar (BASELINE.json north_star; reading S12).

Per DM row, against the oracle row r (fp64) and the GPU row g (fp32):
  TIME     subtract the ORACLE row's mean from both; rel_l2 = |g - r| / |r - mean(r)|  <= 1e-4
           max_abs = max|g - r| / std(r)                                                 <= 1e-3
           mean_err = |mean(g) - mean(r)| / |mean(r)|                                    <= 1e-6
  FOURIER  the same with bin 0 (the DC term, 256x larger than the rest for u8 data) left out of
           the norms and checked separately to 1e-6 relative.
The literal, mean-included numbers are returned too (they are ~256x smaller and would let a
broken phase through).
"""
import numpy as np

REL_L2_TOL = 1e-4
MAX_ABS_TOL = 1e-3
MEAN_TOL = 1e-6


def time_row_errors(got, ref):
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    m = ref.mean()
    r = ref - m
    diff = got - ref
    std = np.sqrt((r * r).mean())
    return {
        "rel_l2": float(np.sqrt((diff * diff).sum() / (r * r).sum())),
        "max_abs": float(np.abs(diff).max() / std),
        "mean_err": float(abs(got.mean() - m) / abs(m)) if m != 0 else float(abs(got.mean())),
        "rel_l2_literal": float(np.sqrt((diff * diff).sum() / (ref * ref).sum())),
    }


def fourier_row_errors(got, ref):
    got = np.asarray(got, dtype=np.complex128)
    ref = np.asarray(ref, dtype=np.complex128)
    diff = got[1:] - ref[1:]
    p = (np.abs(ref[1:]) ** 2)
    rms = np.sqrt(p.mean())
    return {
        "rel_l2": float(np.sqrt((np.abs(diff) ** 2).sum() / p.sum())),
        "max_abs": float(np.abs(diff).max() / rms),
        "mean_err": float(abs(got[0] - ref[0]) / abs(ref[0])) if ref[0] != 0 else float(abs(got[0])),
        "rel_l2_literal": float(np.sqrt((np.abs(got - ref) ** 2).sum() / (np.abs(ref) ** 2).sum())),
    }


def assert_rows(got, ref, mode, what=""):
    """got/ref: [rows][...]; asserts the bar on every row and returns the worst numbers."""
    fn = time_row_errors if mode == "time" else fourier_row_errors
    worst = {"rel_l2": 0.0, "max_abs": 0.0, "mean_err": 0.0, "rel_l2_literal": 0.0}
    for i in range(len(ref)):
        e = fn(got[i], ref[i])
        for k in worst:
            worst[k] = max(worst[k], e[k])
    assert worst["rel_l2"] <= REL_L2_TOL, (what, worst)
    assert worst["max_abs"] <= MAX_ABS_TOL, (what, worst)
    assert worst["mean_err"] <= MEAN_TOL, (what, worst)
    return worst
