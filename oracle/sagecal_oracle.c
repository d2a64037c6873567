/*
 * ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, float64/long-double CPU statement of what the SAGECal
 * direction-dependent calibration hot path computes.  Written from the problem
 * statement (BASELINE.json:5 "north_star"; the paper, PAPER.md, prints no
 * formula -- PAPER.md:25 only says "a single calibration solution will be
 * derived for each cluster") and from the readings listed in SURVEY.md §8(c)
 * and DESIGN.md.  It shares no code, header, table or helper with the CUDA
 * library under paper_1910_13908_b200/ and must never be linked, imported or
 * executed by the product path.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call it.
 *
 * Conventions: N stations, B = N(N-1)/2 baselines in
 * row-major upper-triangle order b(p,q) = p*N - p(p+1)/2 + (q-p-1), p<q;
 * row r = t*B + b; a sample is one 2x2 complex matrix stored row-major
 * [XX, XY, YX, YY]; visibilities [T*B][F][4]; coherencies of one cluster
 * [T*B][F][4]; Jones of one cluster [N][4].
 *
 * No blocking, fusion or reordering beyond the definitions.  Every long sum is
 * accumulated in long double (x87 80-bit) in an order that does not depend on
 * the OpenMP thread count: threads own whole rows / whole baselines, the
 * cross-baseline sums are serial (reading A9).
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): P1-P14 of SURVEY.md §8(c).
 * Parity unpinned: LM constants (tau, Nielsen rule), channel-centre and
 * sigma conventions -- conventions only.
 */
#define _GNU_SOURCE
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex c128;
typedef long double complex c160;

#define C0_M_PER_S 299792458.0L
static const long double TWO_PI_L = 6.283185307179586476925286766559005768L;

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------- */
/* A1-A3: point-source coherencies of ONE cluster.                            */
/*   C[r][c] = sum_s B_s(f_c) exp(-2 pi i (f_c/c0)(u_r l_s + v_r m_s + w_r (n_s-1)))   */
/*   B_s(f) = (f/f0)^alpha_s [[I+Q, U+iV],[U-iV, I-Q]]     (BASELINE.json:5; Q2, Q4, Q5) */
/* n-1 is evaluated as -(l^2+m^2)/(1+sqrt(1-l^2-m^2)) (no cancellation).      */
/* One libm sin/cos per (sample, source); phase reduced in cycles first.      */
/* Q, U, V may be NULL (unpolarised).  rows are independent: any subset of    */
/* uvw rows may be passed.                                                    */
/* ------------------------------------------------------------------------- */
void oracle_predict_cluster(int64_t nrows, int F, const double *freqs, double f0,
                            const double *uvw, int S, const double *l, const double *m,
                            const double *sI, const double *sQ, const double *sU,
                            const double *sV, const double *alpha, c128 *coh) {
    /* loop-invariant per-source quantities (same values as if evaluated in place) */
    long double *nm1 = (long double *)malloc(sizeof(long double) * (size_t)(S > 0 ? S : 1));
    long double *scale = (long double *)malloc(sizeof(long double) * (size_t)(S > 0 ? S : 1) * (size_t)(F > 0 ? F : 1));
    for (int s = 0; s < S; s++) {
        long double ls = l[s], ms = m[s];
        long double r2 = ls * ls + ms * ms;
        nm1[s] = -r2 / (1.0L + sqrtl(1.0L - r2));
        for (int c = 0; c < F; c++)
            scale[(size_t)s * F + c] = powl((long double)freqs[c] / (long double)f0, (long double)alpha[s]);
    }
#pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < nrows; r++) {
        long double u = uvw[3 * r], v = uvw[3 * r + 1], w = uvw[3 * r + 2];
        for (int c = 0; c < F; c++) {
            long double fc = freqs[c];
            c160 acc[4] = {0, 0, 0, 0};
            for (int s = 0; s < S; s++) {
                long double ls = l[s], ms = m[s];
                long double x = (fc / C0_M_PER_S) * (u * ls + v * ms + w * nm1[s]); /* cycles */
                long double xt = x - rintl(x);
                long double ang = TWO_PI_L * xt, sn, cs;
                sincosl(ang, &sn, &cs);
                c160 e = cs - I * sn;
                long double sc = scale[(size_t)s * F + c];
                long double q = sQ ? sQ[s] : 0.0L, uu = sU ? sU[s] : 0.0L, vv = sV ? sV[s] : 0.0L;
                long double ii = sI[s];
                acc[0] += (sc * (ii + q)) * e;
                acc[1] += (sc * (uu + I * vv)) * e;
                acc[2] += (sc * (uu - I * vv)) * e;
                acc[3] += (sc * (ii - q)) * e;
            }
            c128 *o = coh + ((size_t)r * F + c) * 4;
            for (int k = 0; k < 4; k++) o[k] = (c128)acc[k];
        }
    }
    free(nm1); free(scale);
}

/* 2x2 helpers, row-major */
static inline void mm(const c128 *a, const c128 *b, c128 *o) { /* o = a b */
    o[0] = a[0] * b[0] + a[1] * b[2];
    o[1] = a[0] * b[1] + a[1] * b[3];
    o[2] = a[2] * b[0] + a[3] * b[2];
    o[3] = a[2] * b[1] + a[3] * b[3];
}
static inline void mmh(const c128 *a, const c128 *b, c128 *o) { /* o = a b^H */
    o[0] = a[0] * conj(b[0]) + a[1] * conj(b[1]);
    o[1] = a[0] * conj(b[2]) + a[1] * conj(b[3]);
    o[2] = a[2] * conj(b[0]) + a[3] * conj(b[1]);
    o[3] = a[2] * conj(b[2]) + a[3] * conj(b[3]);
}
static inline void mhm(const c128 *a, const c128 *b, c128 *o) { /* o = a^H b */
    o[0] = conj(a[0]) * b[0] + conj(a[2]) * b[2];
    o[1] = conj(a[0]) * b[1] + conj(a[2]) * b[3];
    o[2] = conj(a[1]) * b[0] + conj(a[3]) * b[2];
    o[3] = conj(a[1]) * b[1] + conj(a[3]) * b[3];
}

static inline void bl_stations(int N, int64_t b, int *pp, int *qq) {
    /* inverse of b(p,q): walk the rows of the upper triangle (slow, obvious) */
    int p = 0;
    int64_t left = b;
    while (left >= N - 1 - p) { left -= N - 1 - p; p++; }
    *pp = p;
    *qq = p + 1 + (int)left;
}

/* ------------------------------------------------------------------------- */
/* A4: vis += sign * J_p C J_q^H for ONE cluster (sign -1 subtracts the       */
/* corrupted model, +1 adds it back).  The all-cluster residual is this call  */
/* repeated for k = 0..K-1 in index order.   (BASELINE.json:5 "the            */
/* Jones-corrupted residual V_pq - J_p C_pq J_q^H")                           */
/* ------------------------------------------------------------------------- */
void oracle_corrupt_accumulate(int N, int T, int F, const c128 *coh, const c128 *jones,
                               double sign, c128 *vis) {
    int64_t B = (int64_t)N * (N - 1) / 2;
#pragma omp parallel for schedule(static)
    for (int64_t b = 0; b < B; b++) {
        int p, q;
        bl_stations(N, b, &p, &q);
        const c128 *Jp = jones + 4 * p, *Jq = jones + 4 * q;
        for (int t = 0; t < T; t++)
            for (int c = 0; c < F; c++) {
                size_t o = (((size_t)t * B + b) * F + c) * 4;
                c128 T1[4], Mo[4];
                mm(Jp, coh + o, T1);
                mmh(T1, Jq, Mo);
                for (int k = 0; k < 4; k++) vis[o + k] += sign * Mo[k];
            }
    }
}

/* ------------------------------------------------------------------------- */
/* A5-A6: cost, gradient blocks G_p and per-station J^H J blocks M_p of ONE   */
/* cluster at Jones J against data x:                                         */
/*   E = x - J_p C J_q^H;  phi = sum ||E||_F^2                                */
/*   T1 = J_p C, A = C J_q^H;  G_p += E A^H, G_q += E^H T1;                   */
/*   M_p += A A^H, M_q += T1^H T1.                                            */
/* (BASELINE.json:5 "the cost, and the gradient and per-station-block J^H J   */
/* accumulation over all N(N-1)/2 baselines"; reading Q1: block diagonal.)    */
/* d phi = -2 Re sum_p tr(G_p^H dJ_p).                                        */
/* ------------------------------------------------------------------------- */
typedef struct { long double phi; c160 Gp[4], Gq[4], Mp[4], Mq[4]; } bl_acc;

void oracle_cost_grad_jtj(int N, int T, int F, const c128 *x, const c128 *coh,
                          const c128 *jones, double *cost, c128 *grad, c128 *jtj) {
    int64_t B = (int64_t)N * (N - 1) / 2;
    bl_acc *acc = (bl_acc *)calloc((size_t)B, sizeof(bl_acc));
#pragma omp parallel for schedule(static)
    for (int64_t b = 0; b < B; b++) {
        int p, q;
        bl_stations(N, b, &p, &q);
        const c128 *Jp = jones + 4 * p, *Jq = jones + 4 * q;
        bl_acc a;
        memset(&a, 0, sizeof a);
        for (int t = 0; t < T; t++)
            for (int c = 0; c < F; c++) {
                size_t o = (((size_t)t * B + b) * F + c) * 4;
                const c128 *C = coh + o;
                c128 T1[4], A[4], Mo[4], E[4], t4[4];
                mm(Jp, C, T1);   /* T1 = J_p C     */
                mmh(C, Jq, A);   /* A  = C J_q^H   */
                mm(Jp, A, Mo);   /* model          */
                for (int k = 0; k < 4; k++) {
                    E[k] = x[o + k] - Mo[k];
                    a.phi += (long double)creal(E[k]) * creal(E[k]) + (long double)cimag(E[k]) * cimag(E[k]);
                }
                mmh(E, A, t4);  for (int k = 0; k < 4; k++) a.Gp[k] += t4[k];
                mhm(E, T1, t4); for (int k = 0; k < 4; k++) a.Gq[k] += t4[k];
                mmh(A, A, t4);  for (int k = 0; k < 4; k++) a.Mp[k] += t4[k];
                mhm(T1, T1, t4); for (int k = 0; k < 4; k++) a.Mq[k] += t4[k];
            }
        acc[b] = a;
    }
    /* serial, fixed-order combine over baselines */
    long double phi = 0;
    c160 *G = (c160 *)calloc((size_t)4 * N, sizeof(c160));
    c160 *M = (c160 *)calloc((size_t)4 * N, sizeof(c160));
    int64_t b = 0;
    for (int p = 0; p < N; p++)
        for (int q = p + 1; q < N; q++, b++) {
            phi += acc[b].phi;
            for (int k = 0; k < 4; k++) {
                G[4 * p + k] += acc[b].Gp[k];
                G[4 * q + k] += acc[b].Gq[k];
                M[4 * p + k] += acc[b].Mp[k];
                M[4 * q + k] += acc[b].Mq[k];
            }
        }
    *cost = (double)phi;
    for (int i = 0; i < 4 * N; i++) { grad[i] = (c128)G[i]; jtj[i] = (c128)M[i]; }
    free(acc); free(G); free(M);
}

/* ------------------------------------------------------------------------- */
/* A7: Levenberg-Marquardt for ONE cluster, block-diagonal Gauss-Newton,      */
/* exactly n_lm trial steps, Nielsen damping (readings Q1, Q12-Q14).          */
/*   mu0 = tau * max_p max((M_p)_00, (M_p)_11), nu = 2                         */
/*   dJ_p = G_p (M_p + mu I)^-1;  J' = J + dJ                                  */
/*   pred = sum_p [Re tr(G_p^H dJ_p) + mu ||dJ_p||_F^2]; rho = (phi-phi')/pred */
/*   accept iff pred > 0 and rho > 0 (all finite):                             */
/*       mu *= max(1/3, 1-(2 rho-1)^3), nu = 2                                 */
/*   else mu *= nu, nu *= 2.   mu clamped to [1e-300, 1e300], nu <= 2^60.      */
/* jones is updated in place; *cost is phi at the accepted J.                 */
/* min_abs_rho (may be NULL) receives min |rho| over the decisions (Q18);     */
/* n_accept (may be NULL) the number of accepted steps.                       */
/* ------------------------------------------------------------------------- */
void oracle_lm(int N, int T, int F, const c128 *x, const c128 *coh, c128 *jones, int n_lm,
               double tau, double *cost, double *min_abs_rho, int *n_accept) {
    size_t n4 = (size_t)4 * N;
    c128 *G = malloc(n4 * sizeof(c128)), *M = malloc(n4 * sizeof(c128));
    c128 *Gn = malloc(n4 * sizeof(c128)), *Mn = malloc(n4 * sizeof(c128));
    c128 *Jn = malloc(n4 * sizeof(c128)), *D = malloc(n4 * sizeof(c128));
    double phi, phin;
    oracle_cost_grad_jtj(N, T, F, x, coh, jones, &phi, G, M);
    double mmax = 0;
    for (int p = 0; p < N; p++) {
        mmax = fmax(mmax, creal(M[4 * p]));
        mmax = fmax(mmax, creal(M[4 * p + 3]));
    }
    double mu = tau * mmax, nu = 2.0;
    for (int it = 0; it < n_lm; it++) {
        long double pred_l = 0;
        for (int p = 0; p < N; p++) {
            /* (M_p + mu I)^-1 of the Hermitian 2x2 [[a, b],[conj b, d]] */
            double a = creal(M[4 * p]) + mu, d = creal(M[4 * p + 3]) + mu;
            c128 bb = M[4 * p + 1];
            double det = a * d - (creal(bb) * creal(bb) + cimag(bb) * cimag(bb));
            c128 inv[4] = {d / det, -bb / det, -conj(bb) / det, a / det};
            mm(G + 4 * p, inv, D + 4 * p);
            for (int k = 0; k < 4; k++) {
                c128 g = G[4 * p + k], dd = D[4 * p + k];
                Jn[4 * p + k] = jones[4 * p + k] + dd;
                pred_l += (long double)creal(g) * creal(dd) + (long double)cimag(g) * cimag(dd);
                pred_l += (long double)mu * ((long double)creal(dd) * creal(dd) + (long double)cimag(dd) * cimag(dd));
            }
        }
        double pred = (double)pred_l;
        oracle_cost_grad_jtj(N, T, F, x, coh, Jn, &phin, Gn, Mn);
        double rho = (phi - phin) / pred;
        int ok = isfinite(phin) && isfinite(pred) && isfinite(rho) && pred > 0.0 && rho > 0.0;
        if (min_abs_rho && isfinite(rho) && fabs(rho) < *min_abs_rho) *min_abs_rho = fabs(rho);
        if (ok) {
            memcpy(jones, Jn, n4 * sizeof(c128));
            memcpy(G, Gn, n4 * sizeof(c128));
            memcpy(M, Mn, n4 * sizeof(c128));
            phi = phin;
            double s = 2.0 * rho - 1.0;
            mu *= fmax(1.0 / 3.0, 1.0 - s * s * s);
            nu = 2.0;
            if (n_accept) (*n_accept)++;
        } else {
            mu *= nu;
            nu *= 2.0;
        }
        if (!(mu >= 1e-300)) mu = 1e-300;
        if (mu > 1e300) mu = 1e300;
        if (nu > 0x1p60) nu = 0x1p60;
    }
    *cost = phi;
    free(G); free(M); free(Gn); free(Mn); free(Jn); free(D);
}

/* ------------------------------------------------------------------------- */
/* A8: SAGE-EM over K clusters (readings Q10, Q11, Q15).                      */
/*   R = V - sum_k J_k C_k J_k^H                                              */
/*   for em, for k (fixed order):  x_k = R + J_k C_k J_k^H  (E-step)          */
/*       (J_k, phi_k) = LM(x_k, C_k, J_k)                    (M-step)          */
/*       R = x_k - J_k C_k J_k^H                                               */
/* coh is [K][T*B][F][4]; jones [K][N][4] in/out; residual [T*B][F][4] out.   */
/* cost_trace (may be NULL) has n_em*K+1 entries: ||R||^2 at the start and    */
/* after every M-step.                                                        */
/* ------------------------------------------------------------------------- */
static double frob2(const c128 *a, size_t n) {
    long double s = 0;
    for (size_t i = 0; i < n; i++) s += (long double)creal(a[i]) * creal(a[i]) + (long double)cimag(a[i]) * cimag(a[i]);
    return (double)s;
}

void oracle_sage(int N, int T, int F, int K, const c128 *vis, const c128 *coh, c128 *jones,
                 c128 *residual, int n_em, int n_lm, double tau, double *cost_per_cluster,
                 double *cost_trace, double *min_abs_rho, int *n_accept) {
    size_t B = (size_t)N * (N - 1) / 2, ns = (size_t)T * B * F, n = ns * 4;
    memcpy(residual, vis, n * sizeof(c128));
    for (int k = 0; k < K; k++)
        oracle_corrupt_accumulate(N, T, F, coh + (size_t)k * n, jones + (size_t)k * 4 * N, -1.0, residual);
    if (min_abs_rho) *min_abs_rho = INFINITY;
    if (n_accept) *n_accept = 0;
    int it = 0;
    if (cost_trace) cost_trace[it++] = frob2(residual, n);
    for (int em = 0; em < n_em; em++)
        for (int k = 0; k < K; k++) {
            const c128 *Ck = coh + (size_t)k * n;
            c128 *Jk = jones + (size_t)k * 4 * N;
            oracle_corrupt_accumulate(N, T, F, Ck, Jk, +1.0, residual);       /* residual now holds x_k */
            oracle_lm(N, T, F, residual, Ck, Jk, n_lm, tau, &cost_per_cluster[k], min_abs_rho, n_accept);
            oracle_corrupt_accumulate(N, T, F, Ck, Jk, -1.0, residual);       /* back to R */
            if (cost_trace) cost_trace[it++] = frob2(residual, n);
        }
}
