/*
 * nmf_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct fp64 CPU implementation of the weighted-NMF
 * hot path of arXiv 2309.04623 (section 2, Eq. 1-3), written
 * from the paper.  It shares no code, header, table or helper with the CUDA
 * library under paper_2309_04623_b200/csrc and neither imports the other.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call it.
 *
 * Notation (BASELINE.json orientation; the paper writes V for Omega):
 *   X [N,P] >= 0, Omega [N,P] >= 0 (0 = missing), W [N,K], H [K,P], row-major.
 *
 * The method is an iteration, so the oracle follows it step by step in the
 * paper's order:
 *   Eq. 3, first line :  H <- H o W^T(V o X) / W^T[V o (WH)]
 *   Eq. 3, second line:  W <- W o (V o X)H^T / [V o (WH)]H^T   (with the NEW H, G3)
 * Each output element is accumulated by one thread in index order; there is
 * no blocking, fusion or reordering.  Entries with Omega == 0 are skipped,
 * not multiplied (G5: "treated as missing data and ignored"),
 * and a ratio is num / max(den, 1e-30) (G4).
 *
 * Parity pins for every function here: tests/test_oracle_pins.py (P1-P12).
 * Nothing in this file is "parity unpinned".
 *
 * Build: gcc -O2 -fopenmp -fPIC -shared -o liboracle.so nmf_oracle.c -lm
 */
#include <stddef.h>
#include <stdlib.h>
#include <math.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_EPS 1e-30

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* omega may be NULL (= all ones, SURVEY 8(b) nmf_project) */
static inline double om_at(const float* Om, size_t i) { return Om ? (double)Om[i] : 1.0; }

/* ---- Eq. 3 first line: one H half-step, all columns ------------------- */
/* PAPER.md:48.  Column p of H depends only on column p of X, Omega, H.     */
void oracle_h_step(int N, long P, int K, const float* X, const float* Om,
                   const double* W, double* H) {
#pragma omp parallel
    {
        double* h = (double*)malloc(sizeof(double) * K);
        double* num = (double*)malloc(sizeof(double) * K);
        double* den = (double*)malloc(sizeof(double) * K);
#pragma omp for schedule(static)
        for (long p = 0; p < P; ++p) {
            for (int k = 0; k < K; ++k) { h[k] = H[(size_t)k * P + p]; num[k] = 0.0; den[k] = 0.0; }
            for (int n = 0; n < N; ++n) {
                size_t i = (size_t)n * P + p;
                double om = om_at(Om, i);
                if (!(om > 0.0)) continue;               /* missing datum: ignored */
                double s = 0.0;                          /* (WH)[n,p], old column  */
                for (int k = 0; k < K; ++k) s += W[(size_t)n * K + k] * h[k];
                double q = om * (double)X[i];            /* (V o X)[n,p]           */
                double r = om * s;                       /* (V o WH)[n,p]          */
                for (int k = 0; k < K; ++k) {
                    num[k] += W[(size_t)n * K + k] * q;  /* W^T (V o X)            */
                    den[k] += W[(size_t)n * K + k] * r;  /* W^T [V o (WH)]         */
                }
            }
            for (int k = 0; k < K; ++k)
                H[(size_t)k * P + p] = h[k] * num[k] / fmax(den[k], ORACLE_EPS);
        }
        free(h); free(num); free(den);
    }
}

/* ---- Eq. 3 second line: one W half-step, all rows ---------------------- */
/* PAPER.md:50.  Row n of W depends only on row n of X, Omega, W (and H).    */
void oracle_w_step(int N, long P, int K, const float* X, const float* Om,
                   double* W, const double* H) {
#pragma omp parallel
    {
        double* num = (double*)malloc(sizeof(double) * K);
        double* den = (double*)malloc(sizeof(double) * K);
#pragma omp for schedule(dynamic, 1)
        for (int n = 0; n < N; ++n) {
            double* w = W + (size_t)n * K;
            for (int k = 0; k < K; ++k) { num[k] = 0.0; den[k] = 0.0; }
            for (long p = 0; p < P; ++p) {
                size_t i = (size_t)n * P + p;
                double om = om_at(Om, i);
                if (!(om > 0.0)) continue;
                double s = 0.0;                          /* (WH)[n,p], old row     */
                for (int k = 0; k < K; ++k) s += w[k] * H[(size_t)k * P + p];
                double q = om * (double)X[i];
                double r = om * s;
                for (int k = 0; k < K; ++k) {
                    num[k] += q * H[(size_t)k * P + p];  /* (V o X) H^T            */
                    den[k] += r * H[(size_t)k * P + p];  /* [V o (WH)] H^T         */
                }
            }
            for (int k = 0; k < K; ++k) w[k] = w[k] * num[k] / fmax(den[k], ORACLE_EPS);
        }
        free(num); free(den);
    }
}

/* ---- Eq. 2: weighted Frobenius cost ------------------------------------ */
/* PAPER.md:44.  sum over Omega>0 of Omega*(X - WH)^2.                       */
double oracle_objective(int N, long P, int K, const float* X, const float* Om,
                        const double* W, const double* H) {
    double* rows = (double*)calloc((size_t)N, sizeof(double));
#pragma omp parallel for schedule(dynamic, 1)
    for (int n = 0; n < N; ++n) {
        double f = 0.0;
        for (long p = 0; p < P; ++p) {
            size_t i = (size_t)n * P + p;
            double om = om_at(Om, i);
            if (!(om > 0.0)) continue;
            double s = 0.0;
            for (int k = 0; k < K; ++k) s += W[(size_t)n * K + k] * H[(size_t)k * P + p];
            double d = (double)X[i] - s;
            f += om * d * d;
        }
        rows[n] = f;
    }
    double f = 0.0;
    for (int n = 0; n < N; ++n) f += rows[n];
    free(rows);
    return f;
}

/* ---- the fit: iters x { H half-step ; W half-step } --------------------- */
/* PAPER.md:48-53; fixed iteration count (G7), H first (G2), W sees new H (G3).
 * If trace != NULL it receives 2*iters+1 objective values:
 * f0, then after every H half-step and every W half-step (pin P1).          */
void oracle_fit(int N, long P, int K, const float* X, const float* Om,
                double* W, double* H, int iters, double* trace) {
    if (trace) trace[0] = oracle_objective(N, P, K, X, Om, W, H);
    for (int it = 0; it < iters; ++it) {
        oracle_h_step(N, P, K, X, Om, W, H);
        if (trace) trace[2 * it + 1] = oracle_objective(N, P, K, X, Om, W, H);
        oracle_w_step(N, P, K, X, Om, W, H);
        if (trace) trace[2 * it + 2] = oracle_objective(N, P, K, X, Om, W, H);
    }
}

/* ---- target modelling: non-negative projection on fixed components ------ */
/* PAPER.md:89 "model each target frame individually"; reading G11: the W-type
 * update of Eq. 3 with H frozen, one row per science frame, rows independent. */
void oracle_project(int M, long P, int K, const double* H, const float* T,
                    const float* om_t /* nullable */, double* C, int iters) {
    for (int it = 0; it < iters; ++it) oracle_w_step(M, P, K, T, om_t, C, H);
}

/* ---- PSF subtraction ----------------------------------------------------- */
/* residual = target - model; model = factor * (c . H).
 * Where om_t is given and zero the output is `fill` (G13).                   */
void oracle_subtract(int M, long P, int K, const double* H, const float* T,
                     const double* C, const float* om_t /* nullable */,
                     const double* factor /* [M] nullable = 1 */, double fill, double* out) {
#pragma omp parallel for schedule(static)
    for (long p = 0; p < P; ++p) {
        for (int m = 0; m < M; ++m) {
            size_t i = (size_t)m * P + p;
            if (om_t && !((double)om_t[i] > 0.0)) { out[i] = fill; continue; }
            double s = 0.0;
            for (int k = 0; k < K; ++k) s += C[(size_t)m * K + k] * H[(size_t)k * P + p];
            double f = factor ? factor[m] : 1.0;
            out[i] = (double)T[i] - f * s;
        }
    }
}

/* ---- closest-frame reference selection ------------- */
/* "The target PSFs are then compared to the reference library, and a
 * percentage of the closest frames ... are selected.  The closest frames are
 * calculated by minimizing for Euclidean norm".  Readings (G19, G20):
 *   D[m,n] = sum over the pixels that are valid in BOTH frames (om_t[m,p] > 0 and
 *            Om[n,p] > 0; masked regions are "missing data and ignored",
 *            PAPER.md:81) of (T[m,p] - X[n,p])^2      -- squared Euclidean distance;
 *   the n_sel closest references of target m are the n_sel smallest D[m,:], ties
 *   broken by the lower frame index, listed in ascending order of (D, index).
 * The percentage itself is the caller's choice (the paper gives no formula).
 * Pins: tests/test_oracle_pins.py (brute force, identities, masks, ties).        */
void oracle_ref_distance(int M, int N, long P, const float* T, const float* om_t /* nullable */,
                         const float* X, const float* Om /* nullable */, double* D /* [M,N] */) {
#pragma omp parallel for schedule(static) collapse(2)
    for (int m = 0; m < M; ++m)
        for (int n = 0; n < N; ++n) {
            double s = 0.0;
            for (long p = 0; p < P; ++p) {
                if (om_t && !((double)om_t[(size_t)m * P + p] > 0.0)) continue;
                if (Om && !((double)Om[(size_t)n * P + p] > 0.0)) continue;
                const double d = (double)T[(size_t)m * P + p] - (double)X[(size_t)n * P + p];
                s += d * d;
            }
            D[(size_t)m * N + n] = s;
        }
}

void oracle_ref_select(int M, int N, const double* D, int n_sel, int* idx /* [M,n_sel] */) {
    for (int m = 0; m < M; ++m) {
        const double* d = D + (size_t)m * N;
        for (int n = 0; n < N; ++n) {            /* rank of n under the order (D, index) */
            int rank = 0;
            for (int j = 0; j < N; ++j)
                if (d[j] < d[n] || (d[j] == d[n] && j < n)) ++rank;
            if (rank < n_sel) idx[(size_t)m * n_sel + rank] = n;
        }
    }
}
