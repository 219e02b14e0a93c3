"""Pins of oracle/variants.py (not gpu): the fixed-mean form and the normalisations against things other than
themselves — scipy's own Lomb-Scargle, and weighted least squares with chi2 taken from the residuals."""
import numpy as np
import pytest
from scipy.signal import lombscargle

from oracle import variants


def _series(seed, Nd=57):
    rng = np.random.default_rng(seed)
    t = np.sort(rng.uniform(0, 30, Nd))
    dy = rng.uniform(0.4, 1.6, Nd)
    y = 2.0 + 1.1 * np.sin(2 * np.pi * 0.37 * t + 0.3) + rng.normal(0, 1, Nd) * dy
    return t, y, dy


def _lsq_chi2(t, y, dy, f, offset):
    """chi2 of the best weighted fit of a cos + b sin (+ c) at frequency f, and chi2 of the reference model."""
    w = dy ** -2.0
    ybar = np.sum(w * y) / np.sum(w)
    cols = [np.cos(2 * np.pi * f * t), np.sin(2 * np.pi * f * t)] + ([np.ones_like(t)] if offset else [])
    A = np.stack(cols, 1) / dy[:, None]
    b = (y - (0.0 if offset else ybar)) / dy
    coef, *_ = np.linalg.lstsq(A, b, rcond=None)
    return float(np.sum((A @ coef - b) ** 2)), float(np.sum(((y - ybar) / dy) ** 2))


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_fixed_mean_against_scipy_and_least_squares(seed):
    t, y, dy = _series(seed)
    f0, df, Nf = 0.05, 0.013, 90
    f = f0 + df * np.arange(Nf)
    P = variants.power(t, y, dy, f0, df, Nf, fit_mean=False)
    w = dy ** -2.0
    yc = y - np.sum(w * y) / np.sum(w)
    Ps = lombscargle(t, yc, 2 * np.pi * f, normalize=True, weights=w, floating_mean=False)
    assert np.max(np.abs(P - Ps)) <= 1e-12
    for k in (0, 17, 89):
        chi2, ref = _lsq_chi2(t, y, dy, f[k], offset=False)
        assert abs(P[k] - (1 - chi2 / ref)) <= 1e-12
    # the floating-mean form differs (it fits the offset): the two must not be confused
    assert np.max(np.abs(P - variants.power(t, y, dy, f0, df, Nf, fit_mean=True))) > 1e-4


@pytest.mark.parametrize("fit_mean", [True, False])
def test_normalisations_from_residual_chi2(fit_mean):
    t, y, dy = _series(11)
    f0, df, Nf = 0.05, 0.02, 40
    f = f0 + df * np.arange(Nf)
    got = {n: variants.power(t, y, dy, f0, df, Nf, fit_mean=fit_mean, normalization=n) for n in variants.NORMALIZATIONS}
    for k in (0, 9, 39):
        chi2, ref = _lsq_chi2(t, y, dy, f[k], offset=fit_mean)
        assert abs(got["standard"][k] - (1 - chi2 / ref)) <= 1e-12
        assert abs(got["model"][k] - (ref - chi2) / chi2) <= 1e-11
        assert abs(got["log"][k] - np.log(ref / chi2)) <= 1e-12
        assert abs(got["psd"][k] - 0.5 * (ref - chi2)) <= 1e-10 * ref
    with pytest.raises(ValueError):
        variants.power(t, y, dy, f0, df, Nf, normalization="nope")
