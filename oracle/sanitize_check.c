/*
 * sanitize_check.c -- TEST INFRASTRUCTURE ONLY (ASan / UBSan on the oracle).
 *
 * A tiny driver that calls every function of rmsynth_oracle.c on exactly-sized heap buffers (so that an
 * out-of-bounds index trips AddressSanitizer) with edge shapes: one channel, one depth, a zero-weight channel,
 * a non-finite line of sight, peaks at both grid edges, RM-CLEAN with zero iterations and with a cutoff.
 * tests/test_oracle_sanitizers.py compiles it together with rmsynth_oracle.c under
 *   gcc -fsanitize=address,undefined -fno-sanitize-recover=all
 * and expects exit code 0 and the line "sanitize_check ok".  It checks memory safety and undefined behaviour,
 * not values (the pins do that).
 */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>

void oracle_lambda_sq(const double *nu_hz, int n_chan, double *lam2);
int oracle_plan_scalars(const double *lam2, const double *w, int n_chan, int lambda0_mode, double lambda0_in,
                        double *K_out, double *lambda0_sq_out);
void oracle_rmsf(const double *lam2, const double *w, int n_chan, double K, double lambda0_sq,
                 const double *phi, int n_phi, double *R_re, double *R_im);
void oracle_naive(const float *Q, const float *U, long long n_pix, const double *lam2, const double *w, int n_chan,
                  double K, double lambda0_sq, const double *phi, int n_phi, double *FQ, double *FU);
int oracle_table(const float *Q, const float *U, long long n_pix, const double *lam2, const double *w, int n_chan,
                 double K, double lambda0_sq, const double *phi, int n_phi, double *FQ, double *FU, int n_threads);
void oracle_tolerance_scale(const float *Q, const float *U, long long n_pix, const double *w, int n_chan, double K,
                            double *T);
void oracle_peaks(const double *FQ, const double *FU, long long n_pix, const double *phi, int n_phi,
                  double lambda0_sq, int *kstar, double *peak_amp, double *peak_phi, double *pa_lambda0,
                  double *pa_zero);
void oracle_rmclean(const double *FQ, const double *FU, long long n_pix, int n_phi, const double *Rdw_re,
                    const double *Rdw_im, double gain, double cutoff, int max_iter, double dphi, double fwhm,
                    double *model_q, double *model_u, double *resid_q, double *resid_u, double *rest_q,
                    double *rest_u, int *n_iter, double *min_margin);

static void *xmalloc(size_t n) { void *p = malloc(n ? n : 1); if (!p) exit(2); return p; }

static int run_case(int n_chan, int n_phi, int n_pix, int flag_channel, int nan_pixel)
{
    double *nu = xmalloc(sizeof(double) * n_chan), *w = xmalloc(sizeof(double) * n_chan);
    double *lam2 = xmalloc(sizeof(double) * n_chan), *phi = xmalloc(sizeof(double) * n_phi);
    float *Q = xmalloc(sizeof(float) * n_pix * n_chan), *U = xmalloc(sizeof(float) * n_pix * n_chan);
    for (int i = 0; i < n_chan; ++i) { nu[i] = 1.2e8 + 3.0e5 * i; w[i] = 1.0; }
    if (flag_channel >= 0 && flag_channel < n_chan && n_chan > 1) w[flag_channel] = 0.0;
    for (int k = 0; k < n_phi; ++k) phi[k] = -3.0 + 0.5 * k;
    for (int p = 0; p < n_pix; ++p)
        for (int i = 0; i < n_chan; ++i) {
            Q[p * n_chan + i] = (float)cos(0.3 * i + p);
            U[p * n_chan + i] = (float)sin(0.7 * i - p);
        }
    if (nan_pixel >= 0 && nan_pixel < n_pix) Q[nan_pixel * n_chan] = NAN;
    if (flag_channel >= 0 && flag_channel < n_chan && n_chan > 1)
        for (int p = 0; p < n_pix; ++p) U[p * n_chan + flag_channel] = INFINITY;     /* reading A13: never read */

    oracle_lambda_sq(nu, n_chan, lam2);
    double K = 0.0, l0 = 0.0;
    for (int mode = 0; mode < 3; ++mode)
        if (oracle_plan_scalars(lam2, w, n_chan, mode, 0.25, &K, &l0) != 0) return 1;
    if (oracle_plan_scalars(lam2, w, n_chan, 0, 0.0, &K, &l0) != 0) return 1;

    double *Rre = xmalloc(sizeof(double) * n_phi), *Rim = xmalloc(sizeof(double) * n_phi);
    oracle_rmsf(lam2, w, n_chan, K, l0, phi, n_phi, Rre, Rim);

    size_t nf = (size_t)n_pix * n_phi;
    double *FQ = xmalloc(sizeof(double) * nf), *FU = xmalloc(sizeof(double) * nf);
    double *GQ = xmalloc(sizeof(double) * nf), *GU = xmalloc(sizeof(double) * nf);
    oracle_naive(Q, U, n_pix, lam2, w, n_chan, K, l0, phi, n_phi, FQ, FU);
    if (oracle_table(Q, U, n_pix, lam2, w, n_chan, K, l0, phi, n_phi, GQ, GU, 2) < 0) return 1;   /* returns the number of threads used */
    double *T = xmalloc(sizeof(double) * n_pix);
    oracle_tolerance_scale(Q, U, n_pix, w, n_chan, K, T);

    int *ks = xmalloc(sizeof(int) * n_pix);
    double *amp = xmalloc(sizeof(double) * n_pix), *pp = xmalloc(sizeof(double) * n_pix);
    double *pa0 = xmalloc(sizeof(double) * n_pix), *paz = xmalloc(sizeof(double) * n_pix);
    oracle_peaks(FQ, FU, n_pix, phi, n_phi, l0, ks, amp, pp, pa0, paz);
    /* peaks forced to both grid edges */
    for (int p = 0; p < n_pix; ++p) { GQ[(size_t)p * n_phi] = 1e3; GU[(size_t)p * n_phi + n_phi - 1] = (p & 1) ? 2e3 : 0.0; }
    oracle_peaks(GQ, GU, n_pix, phi, n_phi, l0, ks, amp, pp, pa0, paz);

    /* RM-CLEAN on the double-width grid */
    int m = 2 * n_phi - 1;
    double *ph2 = xmalloc(sizeof(double) * m), *R2r = xmalloc(sizeof(double) * m), *R2i = xmalloc(sizeof(double) * m);
    for (int i = 0; i < m; ++i) ph2[i] = 0.5 * (i - (n_phi - 1));
    oracle_rmsf(lam2, w, n_chan, K, l0, ph2, m, R2r, R2i);
    double *mq = xmalloc(sizeof(double) * nf), *mu = xmalloc(sizeof(double) * nf), *rq = xmalloc(sizeof(double) * nf);
    double *ru = xmalloc(sizeof(double) * nf), *sq = xmalloc(sizeof(double) * nf), *su = xmalloc(sizeof(double) * nf);
    int *nit = xmalloc(sizeof(int) * n_pix);
    double *mm = xmalloc(sizeof(double) * n_pix);
    oracle_rmclean(FQ, FU, n_pix, n_phi, R2r, R2i, 0.1, 0.0, 0, 0.5, 1.5, mq, mu, rq, ru, sq, su, nit, mm);
    oracle_rmclean(FQ, FU, n_pix, n_phi, R2r, R2i, 0.3, 1e-3, 25, 0.5, 1.5, mq, mu, rq, ru, NULL, NULL, nit, mm);
    oracle_rmclean(FQ, FU, n_pix, n_phi, R2r, R2i, 1.0, 1e9, 5, 0.5, 1.5, mq, mu, rq, ru, sq, su, nit, mm);

    free(nu); free(w); free(lam2); free(phi); free(Q); free(U); free(Rre); free(Rim); free(FQ); free(FU); free(GQ);
    free(GU); free(T); free(ks); free(amp); free(pp); free(pa0); free(paz); free(ph2); free(R2r); free(R2i); free(mq);
    free(mu); free(rq); free(ru); free(sq); free(su); free(nit); free(mm);
    return 0;
}

int main(void)
{
    int rc = 0;
    rc |= run_case(1, 1, 1, -1, -1);
    rc |= run_case(2, 2, 3, 0, -1);
    rc |= run_case(7, 13, 5, 3, 2);
    rc |= run_case(33, 9, 4, 32, 0);
    rc |= run_case(16, 3, 2, -1, 1);
    if (rc) { printf("sanitize_check: an oracle call returned an error\n"); return 1; }
    printf("sanitize_check ok\n");
    return 0;
}
