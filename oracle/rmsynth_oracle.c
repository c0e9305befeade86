/*
 * rmsynth_oracle.c -- FP64 CPU oracle for Faraday rotation-measure synthesis.
 *
 * TEST INFRASTRUCTURE ONLY.  This file is the slow, plain, obviously-correct
 * statement of what the CUDA path must compute.  It shares no code, header,
 * table or constant with paper_1810_06250_b200/csrc/.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may load it.
 *
 * Every function cites the passage of /root/reference/PAPER.md (P:L<n>) it
 * follows; readings of silent/garbled passages are the A<n> rows of SURVEY.md
 * section 8(c), restated in DESIGN.md.
 *
 * Pin status (tests/test_oracle_pins.py):
 *   lambda^2, K, lambda0^2, F (naive + table), R, T_p, k*  : pinned (P1-P11, P13)
 *   RM-CLEAN loop (oracle_rmclean, readings C1-C8)         : pinned (C-pins: exact
 *     decomposition identity, geometric series of an on-grid point source, two
 *     separated sources, zero iterations, threshold stop)
 *   parabolic refinement, PA maps (A8-A10)                 : pinned by P12 only
 *     (exact parabola, on-grid point source); the paper prints no worked
 *     example for them -> "parity unpinned" beyond P12.
 *
 * Layout for all cube arguments here: LOS-major, Q[p*n_chan + i],
 * F[p*n_phi + k].  Frequency-major callers transpose before calling.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_C_M_PER_S 299792458.0 /* exact SI value; A1 */

/* P:L117 "measured at lambda_i"; reading A1: lambda_i^2 = (c/nu_i)^2 at the
 * channel centre frequency, nu in Hz. */
void oracle_lambda_sq(const double *nu_hz, int n_chan, double *lam2)
{
    for (int i = 0; i < n_chan; ++i) {
        double lam = ORACLE_C_M_PER_S / nu_hz[i];
        lam2[i] = lam * lam;
    }
}

/* Eq. 13: K = 1 / sum_i w_i.
 * P:L119 "lambda_0^2 ... set to the mean of lambda_i^2"; reading A2:
 *   mode 0: weighted mean K*sum w_i lambda_i^2 (default),
 *   mode 1: plain mean over all channels,
 *   mode 2: the caller's value lambda0_in (0 reproduces Fig. 1 left).
 * Returns 0, or -1 if sum w == 0. */
int oracle_plan_scalars(const double *lam2, const double *w, int n_chan,
                        int lambda0_mode, double lambda0_in,
                        double *K_out, double *lambda0_sq_out)
{
    double W = 0.0, S = 0.0, P = 0.0;
    for (int i = 0; i < n_chan; ++i) {
        W += w[i];
        S += w[i] * lam2[i];
        P += lam2[i];
    }
    if (!(W > 0.0)) return -1;
    *K_out = 1.0 / W;
    if (lambda0_mode == 0) *lambda0_sq_out = S / W;
    else if (lambda0_mode == 1) *lambda0_sq_out = P / (double)n_chan;
    else *lambda0_sq_out = lambda0_in;
    return 0;
}

/* Eq. 12: R(phi) = K sum_i w_i exp(-2 i phi (lambda_i^2 - lambda_0^2)). */
void oracle_rmsf(const double *lam2, const double *w, int n_chan,
                 double K, double lambda0_sq,
                 const double *phi, int n_phi, double *R_re, double *R_im)
{
    for (int k = 0; k < n_phi; ++k) {
        double sr = 0.0, si = 0.0;
        for (int i = 0; i < n_chan; ++i) {
            double th = 2.0 * phi[k] * (lam2[i] - lambda0_sq);
            sr += w[i] * cos(th);
            si -= w[i] * sin(th);
        }
        R_re[k] = K * sr;
        R_im[k] = K * si;
    }
}

/* Eqs. 15-16 / 18-19 with the weights of Eq. 7/11 (reading A3)
 * and the sign of Eq. 11 (A4):
 *   FQ[p,k] = K sum_i w_i ( Q[p,i] cos th_ik + U[p,i] sin th_ik )
 *   FU[p,k] = K sum_i w_i ( U[p,i] cos th_ik - Q[p,i] sin th_ik )
 *   th_ik   = 2 phi_k (lambda_i^2 - lambda_0^2)
 * Literal form: cos/sin evaluated inside the innermost loop, channel order,
 * plain FP64 accumulation.  Q,U are the FP32 samples promoted to FP64 (A12).
 * Reading A13: a channel with w_i = 0 has been REMOVED ("bad channels were
 * removed before processing"): its samples are never read, so whatever
 * a flagged channel holds (NaN-blanked planes included) cannot reach F. */
void oracle_naive(const float *Q, const float *U, long long n_pix,
                  const double *lam2, const double *w, int n_chan,
                  double K, double lambda0_sq,
                  const double *phi, int n_phi, double *FQ, double *FU)
{
    for (long long p = 0; p < n_pix; ++p) {
        for (int k = 0; k < n_phi; ++k) {
            double sq = 0.0, su = 0.0;
            for (int i = 0; i < n_chan; ++i) {
                if (w[i] == 0.0) continue; /* A13 */
                double th = 2.0 * phi[k] * (lam2[i] - lambda0_sq);
                double c = cos(th), s = sin(th);
                double q = (double)Q[p * n_chan + i], u = (double)U[p * n_chan + i];
                sq += w[i] * (q * c + u * s);
                su += w[i] * (u * c - q * s);
            }
            FQ[p * n_phi + k] = K * sq;
            FU[p * n_phi + k] = K * su;
        }
    }
}

/* Same sums as oracle_naive; the only change is that cos/sin of th_ik are
 * evaluated once per (i,k) instead of once per (p,i,k) -- they do not depend
 * on p ("need to computed only once for the entire dataset") -- and
 * the independent lines of sight are spread over OpenMP threads.
 * Returns the number of threads used. */
int oracle_table(const float *Q, const float *U, long long n_pix,
                 const double *lam2, const double *w, int n_chan,
                 double K, double lambda0_sq,
                 const double *phi, int n_phi, double *FQ, double *FU,
                 int n_threads)
{
    size_t nt = (size_t)n_chan * (size_t)n_phi;
    double *C = (double *)malloc(nt * sizeof(double));
    double *S = (double *)malloc(nt * sizeof(double));
    if (!C || !S) { free(C); free(S); return -1; }
    for (int k = 0; k < n_phi; ++k)
        for (int i = 0; i < n_chan; ++i) {
            double th = 2.0 * phi[k] * (lam2[i] - lambda0_sq);
            C[(size_t)k * n_chan + i] = cos(th);
            S[(size_t)k * n_chan + i] = sin(th);
        }
    int used = 1;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#pragma omp parallel
    {
#pragma omp single
        used = omp_get_num_threads();
#pragma omp for schedule(static)
#endif
        for (long long p = 0; p < n_pix; ++p) {
            const float *q = Q + p * n_chan, *u = U + p * n_chan;
            for (int k = 0; k < n_phi; ++k) {
                const double *c = C + (size_t)k * n_chan, *s = S + (size_t)k * n_chan;
                double sq = 0.0, su = 0.0;
                for (int i = 0; i < n_chan; ++i) {
                    if (w[i] == 0.0) continue; /* A13 */
                    double qi = (double)q[i], ui = (double)u[i];
                    sq += w[i] * (qi * c[i] + ui * s[i]);
                    su += w[i] * (ui * c[i] - qi * s[i]);
                }
                FQ[p * n_phi + k] = K * sq;
                FU[p * n_phi + k] = K * su;
            }
        }
#ifdef _OPENMP
    }
#endif
    free(C); free(S);
    return used;
}

/* Tolerance scale of BASELINE.json north_star: T_p = K sum_i w_i |P_i|,
 * |P_i| = sqrt(Q^2+U^2).  By the triangle inequality |F[p,k]| <= T_p. */
void oracle_tolerance_scale(const float *Q, const float *U, long long n_pix,
                            const double *w, int n_chan, double K, double *T)
{
    for (long long p = 0; p < n_pix; ++p) {
        double s = 0.0;
        for (int i = 0; i < n_chan; ++i) {
            if (w[i] == 0.0) continue; /* A13 */
            double q = (double)Q[p * n_chan + i], u = (double)U[p * n_chan + i];
            s += w[i] * sqrt(q * q + u * u);
        }
        T[p] = K * s;
    }
}

/* wrap an angle to [-pi/2, pi/2) (polarisation angles are defined mod pi) */
static double wrap_half_pi(double a)
{
    const double pi = 3.14159265358979323846;
    double r = fmod(a + 0.5 * pi, pi);
    if (r < 0.0) r += pi;
    return r - 0.5 * pi;
}

/* Peak maps.  P:L123: phi_peak is where |F~(phi)| is maximum; Eq. 17
 * |F| = sqrt(FQ^2+FU^2); Eq. 14 (garbled -> reading A9).
 * Readings A8-A10:
 *   k* = lowest index of the maximum of y_k = |F_k|;
 *   3-point parabola through (phi_{k*-1},y-), (phi_{k*},y0), (phi_{k*+1},y+)
 *   on a possibly non-uniform grid (Lagrange form); no refinement at the grid
 *   edges or when the parabola is not strictly concave;
 *   pa_lambda0 = 0.5 atan2(FU_{k*}, FQ_{k*});
 *   pa_zero    = wrap(pa_lambda0 - phi_peak * lambda_0^2) to [-pi/2, pi/2).
 * Reading A17: a line of sight with a non-finite |F| at any depth has no peak:
 *   k* = -1 and NaN in every map.
 */
void oracle_peaks(const double *FQ, const double *FU, long long n_pix,
                  const double *phi, int n_phi, double lambda0_sq,
                  int *kstar, double *peak_amp, double *peak_phi,
                  double *pa_lambda0, double *pa_zero)
{
    for (long long p = 0; p < n_pix; ++p) {
        const double *fq = FQ + p * n_phi, *fu = FU + p * n_phi;
        int kb = 0, finite = 1;
        double yb = -1.0;
        for (int k = 0; k < n_phi; ++k) {
            double y = sqrt(fq[k] * fq[k] + fu[k] * fu[k]);
            if (!isfinite(y)) finite = 0;
            if (y > yb) { yb = y; kb = k; }
        }
        if (!finite) {
            /* Reading A17: "where |F~(phi)| is maximum" has no
             * answer when |F| is not a number at some depth; non-finite samples
             * propagate (rmsynth.h), so the line of sight reports k* = -1 and NaN. */
            kstar[p] = -1;
            peak_amp[p] = peak_phi[p] = pa_lambda0[p] = pa_zero[p] = NAN;
            continue;
        }
        double amp = yb, ph = phi[kb];
        if (kb > 0 && kb < n_phi - 1) {
            double x0 = phi[kb - 1] - phi[kb], x2 = phi[kb + 1] - phi[kb];
            double ym = sqrt(fq[kb - 1] * fq[kb - 1] + fu[kb - 1] * fu[kb - 1]);
            double yp = sqrt(fq[kb + 1] * fq[kb + 1] + fu[kb + 1] * fu[kb + 1]);
            /* y(x) = y0 + b x + a x^2 through (x0,ym), (0,y0), (x2,yp) */
            double d0 = (ym - yb) / x0, d2 = (yp - yb) / x2;
            double a = (d2 - d0) / (x2 - x0);
            double b = d0 - a * x0;
            if (a < 0.0) {
                double xv = -b / (2.0 * a);
                ph = phi[kb] + xv;
                amp = yb + 0.5 * b * xv; /* y0 + b xv + a xv^2 with xv = -b/2a */
            }
        }
        kstar[p] = kb;
        peak_amp[p] = amp;
        peak_phi[p] = ph;
        double pa = 0.5 * atan2(fu[kb], fq[kb]);
        pa_lambda0[p] = pa;
        pa_zero[p] = wrap_half_pi(pa - ph * lambda0_sq);
    }
}

/* ------------------------------------------------------------------------
 * RM-CLEAN per line of sight (scope row NEXT-3).  The paper only NAMES the
 * procedure: "Equation 12 is needed only if one wishes to deconvolve R(phi)
 * from the reconstructed Faraday dispersion function using a procedure called
 * RM-CLEAN (Heald 2009)" (footnote 6).  Every step
 * below is therefore a READING, listed as C1-C8 in DESIGN.md section 2b: a
 * Hogbom CLEAN of the complex dirty spectrum F~(phi_k) with the complex RMSF
 * as the beam ("F~ is equivalent to the dirty image and R to the dirty
 * beam").
 *
 *   C1  the depth grid is uniform, phi_k = phi_0 + k dphi, so the beam centred
 *       on sample j is R((k - j) dphi): R is given on the DOUBLE-WIDTH grid
 *       Rdw[m], m = -(n_phi-1) .. n_phi-1, stored at index m + n_phi - 1
 *       (2 n_phi - 1 complex samples; R(0) = 1 by Eq. 12-13).
 *   C2  residual r <- F~ (complex), model m <- 0 (complex, on the same grid).
 *   C3  each iteration: k* = lowest index of the maximum of |r_k|; stop BEFORE
 *       subtracting if |r_k*| < cutoff (absolute, in the units of F) or if
 *       max_iter iterations have been done.
 *   C4  component c = gain * r_k* (complex); m_k* += c;
 *       r_k -= c * Rdw[k - k*]  for every k (complex multiply).
 *   C5  restored spectrum = sum_j m_j G((k - j) dphi) + r_k with the REAL
 *       Gaussian G(x) = exp(-x^2 / (2 sigma^2)), sigma = fwhm / (2 sqrt(2 ln 2)),
 *       fwhm = the caller's value (the FWHM of |R|).
 *   C6  outputs: model (complex), residual (complex), restored (complex, may be
 *       NULL), number of iterations done, and min_margin = the smallest value,
 *       over the iterations, of |r_k*| - (second largest |r_k|): how close the
 *       arg-max decision ever came to a tie (for parity rules, not part of the
 *       algorithm).
 *   C7  a line of sight with a non-finite sample is left alone: model 0,
 *       residual = input, restored = input, iterations 0 (reading A17).
 *   C8  FP64 throughout; FQ, FU are the FP64 dirty cubes, LOS-major.
 */
void oracle_rmclean(const double *FQ, const double *FU, long long n_pix, int n_phi,
                    const double *Rdw_re, const double *Rdw_im,
                    double gain, double cutoff, int max_iter,
                    double dphi, double fwhm,
                    double *model_q, double *model_u,
                    double *resid_q, double *resid_u,
                    double *rest_q, double *rest_u,
                    int *n_iter, double *min_margin)
{
    const int c0 = n_phi - 1; /* index of R(0) in the double-width array */
    for (long long p = 0; p < n_pix; ++p) {
        const double *fq = FQ + p * n_phi, *fu = FU + p * n_phi;
        double *mq = model_q + p * n_phi, *mu = model_u + p * n_phi;
        double *rq = resid_q + p * n_phi, *ru = resid_u + p * n_phi;
        int finite = 1;
        for (int k = 0; k < n_phi; ++k) {
            mq[k] = 0.0; mu[k] = 0.0;
            rq[k] = fq[k]; ru[k] = fu[k];
            if (!isfinite(fq[k]) || !isfinite(fu[k])) finite = 0;
        }
        int it = 0;
        double margin = INFINITY;
        while (finite && it < max_iter) {
            int kb = 0;
            double yb = -1.0, y2nd = -1.0;
            for (int k = 0; k < n_phi; ++k) {
                double y = sqrt(rq[k] * rq[k] + ru[k] * ru[k]);
                if (y > yb) { y2nd = yb; yb = y; kb = k; }
                else if (y > y2nd) y2nd = y;
            }
            if (yb < cutoff) break;                              /* C3 */
            if (n_phi > 1 && yb - y2nd < margin) margin = yb - y2nd;
            double cq = gain * rq[kb], cu = gain * ru[kb];       /* C4 */
            mq[kb] += cq; mu[kb] += cu;
            for (int k = 0; k < n_phi; ++k) {
                double br = Rdw_re[c0 + k - kb], bi = Rdw_im[c0 + k - kb];
                rq[k] -= cq * br - cu * bi;
                ru[k] -= cq * bi + cu * br;
            }
            ++it;
        }
        n_iter[p] = it;
        if (min_margin) min_margin[p] = margin;
        if (rest_q && rest_u) {                                  /* C5 */
            const double sigma = fwhm / (2.0 * sqrt(2.0 * log(2.0)));
            for (int k = 0; k < n_phi; ++k) {
                double sq = rq[k], su = ru[k];
                for (int j = 0; j < n_phi; ++j) {
                    if (mq[j] == 0.0 && mu[j] == 0.0) continue;
                    double x = (double)(k - j) * dphi;
                    double g = exp(-x * x / (2.0 * sigma * sigma));
                    sq += mq[j] * g; su += mu[j] * g;
                }
                rest_q[p * n_phi + k] = sq; rest_u[p * n_phi + k] = su;
            }
        }
    }
}
