/*
 * ls_oracle.c — CPU ORACLE for the floating-mean, weighted, standard-normalised Lomb-Scargle
 * periodogram.  THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code, header,
 * table or constant with the CUDA path (paper_2409_08090_b200/csrc) and never calls it.
 *
 * What it computes is the PLAIN DEFINITION the NUFFT path approximates:
 *   Eq. 1 (§1):  S_k = sum_j h_j sin(2 pi f_k t_j),  C_k = sum_j h_j cos(2 pi f_k t_j)
 * evaluated directly, O(N_d N_f), at f_k = f0 + k df, k = 0..N_f-1 (reading A1),
 * for the weights h_j = w_j (y_j - ybar_w) and w_j at f_k, and w_j at 2 f_k (BASELINE.json north_star;
 * six sums, reading A5), followed by the tau / YY,YC,YS,CC,SS / standard-normalisation
 * assembly named by north_star (the paper cites PR89 / VanderPlas 2018 for it).
 *
 * Steps (SURVEY.md §8(c) O1..O6, O-alt, O-fast):
 *   O1  w_j = dy_j^-2 / sum dy^-2                       (Neumaier-compensated sum)
 *   O2  ybar = sum w_j y_j;  h_j = w_j (y_j - ybar);  YY = sum w_j (y_j - ybar)^2
 *   O3  f_k = f0 + k df held as a double-double (the real number the doubles f0, df define)
 *   O4  phase in cycles frac(f_k t_j) by an FMA two-product;  sincos(2 pi phase)
 *   O5  six Neumaier-compensated sums  Sh, Ch, S, C, S2, C2
 *   O6  assembly -> P_k ; also the tau-free form for an internal cross-check
 *   O-alt  ls_oracle_chi2: 3-parameter weighted least squares a cos + b sin + c on UNCENTRED y,
 *          P = 1 - chi2_min / chi2_0        (the definition of the floating-mean periodogram)
 *   O-fast ls_oracle_winding: the paper's own reference method, "exact angle-sum trigonometric
 *          identities ... (a 'phase winding' method)", re-seeded from O4 every R steps.
 *
 * Precision: fp64 throughout (the paper restricts itself to double); inputs given in
 * fp32 are promoted exactly by the caller.  No blocking, fusion or reordering beyond the above.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): worked example at 50 digits (tests/golden/),
 * scipy.signal.lombscargle, chi2 definition vs tau formulas, equispaced t -> DFT + Parseval,
 * noiseless sinusoid -> P = 1 at its frequency, time-shift and dy-scale invariance, mpmath brute
 * force on N_d <= 64.  Parity unpinned: the conventions for f_k = 0 and exact 0/0 in tan(2 omega tau)
 * (reading A14) — not reachable from the five configs.
 *
 * Build: gcc -O2 -fopenmp -mfma -ffp-contract=off -shared -fPIC  (see oracle/build.py).
 */
#define _GNU_SOURCE   /* sincos() */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define TWO_PI 6.283185307179586476925286766559

/* Neumaier's compensated summation: (s, c) accumulates x; result is s + c. */
static inline void nsum(double *s, double *c, double x) {
    double t = *s + x;
    if (fabs(*s) >= fabs(x)) *c += (*s - t) + x;
    else                     *c += (x - t) + *s;
    *s = t;
}

/* O3: f_k = f0 + k*df as a double-double (hi, lo): error-free product k*df (FMA) + two-sum with f0. */
static inline void freq_dd(double f0, double df, int64_t k, double *hi, double *lo) {
    double kd = (double)k;                 /* exact for k < 2^53 */
    double p = kd * df;
    double pe = fma(kd, df, -p);           /* k*df = p + pe exactly */
    double s = f0 + p;
    double bb = s - f0;
    double se = (f0 - (s - bb)) + (p - bb);/* f0 + p = s + se exactly */
    double l = se + pe;
    double h = s + l;
    *lo = l - (h - s);
    *hi = h;
}

/* O4: phase of f*t in cycles, reduced to [-0.5, 0.5], with an FMA two-product. */
static inline double phase_cycles(double fhi, double flo, double t) {
    double p = fhi * t;
    double e = fma(fhi, t, -p) + flo * t;  /* f*t = p + e (+ O(eps^2)) */
    double r = p - rint(p);                /* exact */
    double ph = r + e;
    return ph - rint(ph);
}

int ls_oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* O1 + O2.  wn[j] = normalised weights, h[j] = wn_j (y_j - ybar); stats = {W, ybar, YY}. */
static void weights_and_centre(int64_t Nd, const double *y, const double *dy,
                               double *wn, double *h, double stats[3]) {
    double s = 0, c = 0;
    for (int64_t j = 0; j < Nd; ++j) { wn[j] = 1.0 / (dy[j] * dy[j]); nsum(&s, &c, wn[j]); }
    double W = s + c;
    for (int64_t j = 0; j < Nd; ++j) wn[j] /= W;
    s = 0; c = 0;
    for (int64_t j = 0; j < Nd; ++j) nsum(&s, &c, wn[j] * y[j]);
    double ybar = s + c;
    s = 0; c = 0;
    for (int64_t j = 0; j < Nd; ++j) {
        double yc = y[j] - ybar;
        h[j] = wn[j] * yc;
        nsum(&s, &c, wn[j] * yc * yc);
    }
    stats[0] = W; stats[1] = ybar; stats[2] = s + c;
}

int ls_oracle_stats(int64_t Nd, const double *y, const double *dy, double *stats /*[3]*/) {
    double *wn = (double *)malloc(sizeof(double) * (size_t)Nd), *h = (double *)malloc(sizeof(double) * (size_t)Nd);
    if (!wn || !h) { free(wn); free(h); return 2; }
    weights_and_centre(Nd, y, dy, wn, h, stats);
    free(wn); free(h);
    return 0;
}

/* O6: assembly.  sums = {Sh, Ch, S, C, S2, C2}.  Returns P; aux[0] = tan(2 omega tau),
 * aux[1] = the tau-free form (must agree with P except where ill-conditioned).
 *   tan 2wt = (S2 - 2 S C) / (C2 - (C^2 - S^2))
 *   C2w = 1/sqrt(1+tan^2),  S2w = tan C2w            [written as |den|/r, num sign(den)/r, r = hypot]
 *   Cw = sqrt((1+C2w)/2),   Sw = sign(S2w) sqrt((1-C2w)/2)   [written as S2w/(2 Cw): same number,
 *                                                             no cancellation when C2w -> 1]
 *   YC = Ch Cw + Sh Sw,  YS = Sh Cw - Ch Sw
 *   CC = (1 + C2 C2w + S2 S2w)/2 - (C Cw + S Sw)^2
 *   SS = (1 - C2 C2w - S2 S2w)/2 - (S Cw - C Sw)^2
 *   P = (YC^2/CC + YS^2/SS) / YY
 * Conventions where the formulas are 0/0 (A14, unpinned): num = den = 0 -> tau = 0;
 * a term whose denominator CC or SS is <= 0 is dropped. */
static double assemble(const double sums[6], double YY, double *aux) {
    double Sh = sums[0], Ch = sums[1], S = sums[2], C = sums[3], S2 = sums[4], C2 = sums[5];
    double num = S2 - 2.0 * S * C;
    double den = C2 - (C * C - S * S);
    double r = hypot(num, den);
    double C2w, S2w;
    if (r == 0.0) { C2w = 1.0; S2w = 0.0; }
    else { C2w = fabs(den) / r; S2w = (den < 0 ? -num : num) / r; }
    double Cw = sqrt(0.5 * (1.0 + C2w));
    double Sw = S2w / (2.0 * Cw);
    double YC = Ch * Cw + Sh * Sw;
    double YS = Sh * Cw - Ch * Sw;
    double a = C * Cw + S * Sw, b = S * Cw - C * Sw;
    double CC = 0.5 * (1.0 + C2 * C2w + S2 * S2w) - a * a;
    double SS = 0.5 * (1.0 - C2 * C2w - S2 * S2w) - b * b;
    double P = 0.0;
    if (CC > 0.0) P += YC * YC / CC;
    if (SS > 0.0) P += YS * YS / SS;
    P /= YY;
    if (aux) {
        aux[0] = (den != 0.0) ? num / den : (num == 0.0 ? 0.0 : copysign(INFINITY, num));
        double CCp = 0.5 * (1.0 + C2) - C * C, SSp = 0.5 * (1.0 - C2) - S * S, CSp = 0.5 * S2 - C * S;
        double D = CCp * SSp - CSp * CSp;
        aux[1] = (SSp * Ch * Ch + CCp * Sh * Sh - 2.0 * CSp * Ch * Sh) / (YY * D);
    }
    return P;
}

/* Direct evaluation (O1..O6).  kidx == NULL -> k = 0..K-1, else the K indices given.
 * variant 0 ("strict"): (s2, c2) from a second sincos at frac(2 phase);
 * variant 1 ("double-angle"): s2 = 2 s c, c2 = 1 - 2 s^2.
 * power[K]; sums (may be NULL) [K][6] = Sh,Ch,S,C,S2,C2; aux (may be NULL) [K][2] = tan2wt, P_taufree. */
int ls_oracle_direct(int64_t Nd, const double *t, const double *y, const double *dy,
                     double f0, double df, int64_t K, const int64_t *kidx, int variant,
                     double *power, double *sums, double *aux) {
    if (Nd < 1 || K < 0) return 1;
    double *wn = (double *)malloc(sizeof(double) * (size_t)Nd), *h = (double *)malloc(sizeof(double) * (size_t)Nd);
    if (!wn || !h) { free(wn); free(h); return 2; }
    double stats[3];
    weights_and_centre(Nd, y, dy, wn, h, stats);
    const double YY = stats[2];
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t q = 0; q < K; ++q) {
        int64_t k = kidx ? kidx[q] : q;
        double fhi, flo;
        freq_dd(f0, df, k, &fhi, &flo);
        double a[6] = {0, 0, 0, 0, 0, 0}, c[6] = {0, 0, 0, 0, 0, 0};
        for (int64_t j = 0; j < Nd; ++j) {
            double ph = phase_cycles(fhi, flo, t[j]);
            double s, co, s2, c2;
            sincos(TWO_PI * ph, &s, &co);
            if (variant == 0) {
                double ph2 = 2.0 * ph; ph2 -= rint(ph2);
                sincos(TWO_PI * ph2, &s2, &c2);
            } else { s2 = 2.0 * s * co; c2 = 1.0 - 2.0 * s * s; }
            nsum(&a[0], &c[0], h[j] * s);   nsum(&a[1], &c[1], h[j] * co);
            nsum(&a[2], &c[2], wn[j] * s);  nsum(&a[3], &c[3], wn[j] * co);
            nsum(&a[4], &c[4], wn[j] * s2); nsum(&a[5], &c[5], wn[j] * c2);
        }
        double sm[6];
        for (int i = 0; i < 6; ++i) sm[i] = a[i] + c[i];
        power[q] = assemble(sm, YY, aux ? aux + 2 * q : NULL);
        if (sums) memcpy(sums + 6 * q, sm, sizeof sm);
    }
    free(wn); free(h);
    return 0;
}

/* O-alt: the definition.  At each f solve min_{a,b,c} sum_j w_j (y_j - a cos - b sin - c)^2 on the
 * UNCENTRED y (normal equations, Gaussian elimination with partial pivoting), evaluate chi2_min as
 * the residual sum in a second pass, P = 1 - chi2_min/chi2_0, chi2_0 = sum w (y - ybar)^2. */
int ls_oracle_chi2(int64_t Nd, const double *t, const double *y, const double *dy,
                   double f0, double df, int64_t K, const int64_t *kidx, double *power) {
    if (Nd < 1 || K < 0) return 1;
    double *wn = (double *)malloc(sizeof(double) * (size_t)Nd), *h = (double *)malloc(sizeof(double) * (size_t)Nd);
    if (!wn || !h) { free(wn); free(h); return 2; }
    double stats[3];
    weights_and_centre(Nd, y, dy, wn, h, stats);
    const double chi0 = stats[2];
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t q = 0; q < K; ++q) {
        int64_t k = kidx ? kidx[q] : q;
        double fhi, flo;
        freq_dd(f0, df, k, &fhi, &flo);
        double A[3][4]; double Ac[3][4];
        memset(A, 0, sizeof A); memset(Ac, 0, sizeof Ac);
        for (int64_t j = 0; j < Nd; ++j) {
            double s, co;
            sincos(TWO_PI * phase_cycles(fhi, flo, t[j]), &s, &co);
            double b[3] = {co, s, 1.0};
            for (int r = 0; r < 3; ++r) {
                for (int cc = 0; cc < 3; ++cc) nsum(&A[r][cc], &Ac[r][cc], wn[j] * b[r] * b[cc]);
                nsum(&A[r][3], &Ac[r][3], wn[j] * b[r] * y[j]);
            }
        }
        double M[3][4];
        for (int r = 0; r < 3; ++r) for (int cc = 0; cc < 4; ++cc) M[r][cc] = A[r][cc] + Ac[r][cc];
        for (int p = 0; p < 3; ++p) {
            int piv = p;
            for (int r = p + 1; r < 3; ++r) if (fabs(M[r][p]) > fabs(M[piv][p])) piv = r;
            if (piv != p) for (int cc = 0; cc < 4; ++cc) { double tmp = M[p][cc]; M[p][cc] = M[piv][cc]; M[piv][cc] = tmp; }
            for (int r = p + 1; r < 3; ++r) {
                double fct = M[r][p] / M[p][p];
                for (int cc = p; cc < 4; ++cc) M[r][cc] -= fct * M[p][cc];
            }
        }
        double x[3];
        for (int p = 2; p >= 0; --p) {
            double v = M[p][3];
            for (int cc = p + 1; cc < 3; ++cc) v -= M[p][cc] * x[cc];
            x[p] = v / M[p][p];
        }
        double rs = 0, rc = 0;
        for (int64_t j = 0; j < Nd; ++j) {
            double s, co;
            sincos(TWO_PI * phase_cycles(fhi, flo, t[j]), &s, &co);
            double res = y[j] - (x[0] * co + x[1] * s + x[2]);
            nsum(&rs, &rc, wn[j] * res * res);
        }
        power[q] = 1.0 - (rs + rc) / chi0;
    }
    free(wn); free(h);
    return 0;
}

/* O-fast: phase winding over the contiguous range k = k0 .. k0+K-1.  Per point the
 * phasor e^{2 pi i f_k t_j} is advanced by the exact angle-sum identity with e^{2 pi i df t_j};
 * it is re-seeded from the double-double phase (O4) every R steps to bound the drift; the 2f sums use
 * the double-angle identities.  Each thread owns a contiguous block of frequencies and its own
 * phasor arrays.  Used for the timed CPU baseline and full-grid sweeps. */
int ls_oracle_winding(int64_t Nd, const double *t, const double *y, const double *dy,
                      double f0, double df, int64_t k0, int64_t K, int R, double *power) {
    if (Nd < 1 || K < 0 || R < 1) return 1;
    double *wn = (double *)malloc(sizeof(double) * (size_t)Nd), *h = (double *)malloc(sizeof(double) * (size_t)Nd);
    double *ds = (double *)malloc(sizeof(double) * (size_t)Nd), *dc = (double *)malloc(sizeof(double) * (size_t)Nd);
    if (!wn || !h || !ds || !dc) { free(wn); free(h); free(ds); free(dc); return 2; }
    double stats[3];
    weights_and_centre(Nd, y, dy, wn, h, stats);
    const double YY = stats[2];
    for (int64_t j = 0; j < Nd; ++j) sincos(TWO_PI * phase_cycles(df, 0.0, t[j]), &ds[j], &dc[j]);
    int fail = 0;
#pragma omp parallel
    {
        double *ps = (double *)malloc(sizeof(double) * (size_t)Nd), *pc = (double *)malloc(sizeof(double) * (size_t)Nd);
        if (!ps || !pc) {
#pragma omp atomic write
            fail = 1;
        } else {
#pragma omp for schedule(static)
            for (int64_t blk = 0; blk < (K + R - 1) / R; ++blk) {
                int64_t qa = blk * R, qb = qa + R < K ? qa + R : K;
                double fhi, flo;
                freq_dd(f0, df, k0 + qa, &fhi, &flo);
                for (int64_t j = 0; j < Nd; ++j) sincos(TWO_PI * phase_cycles(fhi, flo, t[j]), &ps[j], &pc[j]);
                for (int64_t q = qa; q < qb; ++q) {
                    double a[6] = {0, 0, 0, 0, 0, 0}, c[6] = {0, 0, 0, 0, 0, 0};
                    for (int64_t j = 0; j < Nd; ++j) {
                        double s = ps[j], co = pc[j];
                        nsum(&a[0], &c[0], h[j] * s);   nsum(&a[1], &c[1], h[j] * co);
                        nsum(&a[2], &c[2], wn[j] * s);  nsum(&a[3], &c[3], wn[j] * co);
                        nsum(&a[4], &c[4], wn[j] * (2.0 * s * co)); nsum(&a[5], &c[5], wn[j] * (1.0 - 2.0 * s * s));
                        ps[j] = s * dc[j] + co * ds[j];     /* sin(a+b) */
                        pc[j] = co * dc[j] - s * ds[j];     /* cos(a+b) */
                    }
                    double sm[6];
                    for (int i = 0; i < 6; ++i) sm[i] = a[i] + c[i];
                    power[q] = assemble(sm, YY, NULL);
                }
            }
        }
        free(ps); free(pc);
    }
    free(wn); free(h); free(ds); free(dc);
    return fail ? 2 : 0;
}

/* Assembly alone (O6) from given sums: lets tests pin `assemble` against independent values. */
int ls_oracle_assemble(int64_t K, const double *sums /*[K][6]*/, double YY, double *power, double *aux) {
    for (int64_t q = 0; q < K; ++q) power[q] = assemble(sums + 6 * q, YY, aux ? aux + 2 * q : NULL);
    return 0;
}
