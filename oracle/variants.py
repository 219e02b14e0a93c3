"""CPU oracle for the periodogram VARIANTS — TEST INFRASTRUCTURE ONLY, like the rest
of oracle/: the fixed-mean form the paper's abstract describes ("four weighted trigonometric sums", a pair
of NUFFTs, PAPER.md:17 — Press & Rybicki 1989) and the normalisations of the Astropy interface the paper
plugs into (definitions: VanderPlas 2018, which the paper cites).

Plain numpy fp64 on top of the direct sums of ls_oracle.c (Eq. 1):

  fit_mean = True   floating mean, six sums (the default path; power from ls_oracle.c itself)
  fit_mean = False  y centred by its weighted mean, model a cos + b sin WITHOUT an offset: the (S, C) sums of the
                    weights drop out of tau, CC and SS:
                        tan 2 omega tau = S2 / C2
                        YC = Ch cos(wt) + Sh sin(wt),  YS = Sh cos(wt) - Ch sin(wt)
                        CC = (1 + C2 cos 2wt + S2 sin 2wt)/2,  SS = (1 - C2 cos 2wt - S2 sin 2wt)/2
                        P_standard = (YC^2/CC + YS^2/SS) / YY
  normalisation     with chi2_ref = sum ((y - ybar)/dy)^2 = W YY and chi2 the best-fit residual,
                    P_standard = 1 - chi2/chi2_ref:
                        standard  P
                        model     (chi2_ref - chi2)/chi2       = P / (1 - P)
                        log       ln(chi2_ref / chi2)          = -ln(1 - P)
                        psd       (chi2_ref - chi2)/2          = P W YY / 2

Pins: tests/test_oracle_variants.py (scipy.signal.lombscargle with floating_mean=False; weighted least squares
with and without the offset column, chi2 computed from residuals)."""
from __future__ import annotations

import numpy as np

from . import direct, stats

NORMALIZATIONS = ("standard", "model", "log", "psd")


def normalise(P_standard, YY, W, normalization):
    P = np.asarray(P_standard, dtype=np.float64)
    if normalization == "standard":
        return P.copy()
    if normalization == "model":
        return P / (1.0 - P)
    if normalization == "log":
        return -np.log(1.0 - P)
    if normalization == "psd":
        return 0.5 * P * W * YY
    raise ValueError(f"unknown normalization {normalization!r}")


def power(t, y, dy, f0, df, Nf, k=None, fit_mean=True, normalization="standard"):
    """Periodogram of one series at f0 + k df (k default 0..Nf-1) for the chosen variant."""
    W, _, YY = stats(y, dy)
    P, sums, _ = direct(t, y, dy, f0, df, Nf, k=k, return_sums=True)
    if not fit_mean:
        Sh, Ch, S2, C2 = sums[:, 0], sums[:, 1], sums[:, 4], sums[:, 5]
        wt2 = np.arctan2(S2, C2)                     # 2 omega tau
        cw, sw = np.cos(0.5 * wt2), np.sin(0.5 * wt2)
        YC = Ch * cw + Sh * sw
        YS = Sh * cw - Ch * sw
        CC = 0.5 * (1.0 + C2 * np.cos(wt2) + S2 * np.sin(wt2))
        SS = 0.5 * (1.0 - C2 * np.cos(wt2) - S2 * np.sin(wt2))
        P = (YC * YC / CC + YS * YS / SS) / YY
    return normalise(P, YY, W, normalization)
