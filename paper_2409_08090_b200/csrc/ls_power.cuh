// ls_power.cuh — K6 arithmetic shared by the assembly kernels (ls_post.cu) and the FFT pass that is fused
// with the assembly (ls_fft.cu).  Device-only, header-only; internal to libls_b200.so.
#pragma once

#include "../../include/ls.h"

namespace lsb {

// The assembly formulas exactly as north_star lists them, with
//   C2w = |den|/r, S2w = num sign(den)/r, r = hypot(num, den)   [= 1/sqrt(1+tan^2), tan C2w]
//   Sw  = S2w / (2 Cw)                                           [= sign(S2w) sqrt((1-C2w)/2)]
// and the conventions of reading A14 for 0/0 and non-positive CC, SS.
// Per-frequency part (depends on the weights only: shared by every series of a batch with common dy):
// the rotation (Cw, Sw) = (cos, sin)(omega tau) and the reciprocals of CC, SS (0 where the term is dropped).
struct FreqTerms {
    double Cw, Sw, iCC, iSS;                         // rotation, and 1/CC, 1/SS (0 where the term is dropped, A14)
};
// Two reciprocal square roots and one division: 1/r = rsqrt(num^2 + den^2), 1/Cw = rsqrt((1 + C2w)/2)
// (the fp64 sqrt and division sequences were half of this kernel's fp64 work, profiles/r1c_cfg3.md).
__device__ __forceinline__ FreqTerms freq_terms(double S, double C, double S2, double C2) {
    const double num = S2 - 2.0 * S * C;
    const double den = C2 - (C * C - S * S);
    const double r2 = num * num + den * den;
    double C2w = 1.0, S2w = 0.0;                     // tau = 0 when numerator = denominator = 0 (A14)
    if (r2 > 0.0) {
        const double ir = rsqrt(r2);
        C2w = fabs(den) * ir;
        S2w = (den < 0.0 ? -num : num) * ir;
    }
    const double cw2 = 0.5 * (1.0 + C2w);            // in [1/2, 1]
    const double icw = rsqrt(cw2);
    FreqTerms f;
    f.Cw = cw2 * icw;
    f.Sw = 0.5 * S2w * icw;
    const double a = C * f.Cw + S * f.Sw, b = S * f.Cw - C * f.Sw;
    const double CC = 0.5 * (1.0 + C2 * C2w + S2 * S2w) - a * a;
    const double SS = 0.5 * (1.0 - C2 * C2w - S2 * S2w) - b * b;
    if (CC > 0.0 && SS > 0.0) {                      // the usual case: ONE division for both reciprocals
        const double inv = 1.0 / (CC * SS);
        f.iCC = SS * inv;
        f.iSS = CC * inv;
    } else {
        f.iCC = CC > 0.0 ? 1.0 / CC : 0.0;
        f.iSS = SS > 0.0 ? 1.0 / SS : 0.0;
    }
    return f;
}
// Per-series part: YC, YS in the rotated frame and the standard-normalised power (YC^2/CC + YS^2/SS)/YY.
__device__ __forceinline__ double series_power(const FreqTerms& f, double Sh, double Ch, double inv_YY) {
    const double YC = Ch * f.Cw + Sh * f.Sw;
    const double YS = Sh * f.Cw - Ch * f.Sw;
    return (YC * YC * f.iCC + YS * YS * f.iSS) * inv_YY;
}
// Normalisations of the standard power P = 1 - chi2/chi2_ref (VanderPlas 2018, cited PAPER.md:117; the
// Astropy interface the paper plugs into): model P/(1-P), log -ln(1-P), psd P W YY / 2
// (W = sum dy^-2, YY = weighted variance: W YY = chi2_ref).
__device__ __forceinline__ double apply_normalization(double P, int norm, double YY, double W) {
    if (norm == LS_NORM_MODEL) return P / (1.0 - P);
    if (norm == LS_NORM_LOG) return -log(1.0 - P);
    if (norm == LS_NORM_PSD) return 0.5 * P * W * YY;
    return P;
}
__device__ __forceinline__ double assemble_power(double Sh, double Ch, double S, double C, double S2, double C2,
                                                 double inv_YY) {
    return series_power(freq_terms(S, C, S2, C2), Sh, Ch, inv_YY);
}

}  // namespace lsb
