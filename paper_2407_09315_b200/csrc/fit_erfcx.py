"""Generator of the coefficients of sr_erfcx_poly (sr_kernels.cuh): a degree-8 polynomial c(t) with
    erfc(x) = t * c(t) * exp(-x^2),   t = 1 / (1 + x / 2),   0 <= x <= 10,
fitted by weighted least squares for RELATIVE error at Chebyshev nodes in t (so that far pairs, where
erfc is tiny, are as accurate as near ones).  Prints the C array; max relative error with fp32 Horner
evaluation is 3.1e-7.  Not used at run time; run `python fit_erfcx.py` to regenerate."""
import numpy as np
from scipy.special import erfcx

P_, DEG, XMAX = 0.5, 8, 10.0


def fit():
    tmin = 1.0 / (1.0 + P_ * XMAX)
    n = 4000
    t = 0.5 * (1 + tmin) + 0.5 * (1 - tmin) * np.cos(np.pi * (np.arange(n) + 0.5) / n)
    x = (1.0 / t - 1.0) / P_
    f = erfcx(x) / t
    V = np.vander(t, DEG + 1, increasing=True)
    coef, *_ = np.linalg.lstsq(V / f[:, None], np.ones(n), rcond=None)
    return coef


def max_rel_error_fp32(coef):
    xs = np.linspace(0, XMAX, 400001)
    ts = (np.float32(1.0) / (np.float32(1.0) + np.float32(P_) * xs.astype(np.float32))).astype(np.float32)
    acc = np.full_like(ts, np.float32(coef[-1]))
    for c in coef[-2::-1]:
        acc = (acc * ts + np.float32(c)).astype(np.float32)
    return float((np.abs(acc.astype(np.float64) * ts - erfcx(xs)) / erfcx(xs)).max())


if __name__ == "__main__":
    c = fit()
    print("// c_0 .. c_%d (fit_erfcx.py), max relative error %.2e in fp32" % (DEG, max_rel_error_fp32(c)))
    print("{" + ", ".join("%.9ef" % v for v in c) + "}")
