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
 * Parity pins for every function here: tests/test_oracle_pins.py (P1-P24).
 * "Parity unpinned": only the CONVENTIONS of oracle_derotate_stack (rotation centre,
 * bilinear interpolation, mean combination: readings G22-G24 -- the paper states none,
 * PAPER.md:89, 99); the arithmetic those readings define is pinned (P20-P23).  The
 * stopping quantity of oracle_fit_tol is likewise a reading (G21; PAPER.md:53 names no
 * quantity); the function is pinned to that reading (P17-P19).
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

/* ---- tolerance-based stopping ---------------------------------- */
/* the iteration is "left to continue until the change in gradient from one
 * step to the next reaches a set value or the maximum number of iterations is reached".
 * Neither the quantity nor the value is defined in the paper.  Reading G21:
 * the monitored quantity is the cost of Eq. 2, f_t, evaluated after every
 * `check_every` iterations (check_every = 1: "from one step to the next"); the fit stops
 * at the first check t with  |f_{t-check_every} - f_t| < tol * f_{t-check_every}
 * (relative change of the cost between consecutive checks, strict inequality: tol = 0
 * never stops and gives the fixed-count fit), else after max_iters iterations.
 * Returns the number of iterations done; *f_last = cost at the last check (or f_0);
 * trace (nullable) receives f_0 and the cost at every check.
 * Pins: tests/test_oracle_pins.py P17-P19.                                               */
int oracle_fit_tol(int N, long P, int K, const float* X, const float* Om, double* W, double* H,
                   int max_iters, int check_every, double tol, double* f_last, double* trace) {
    double f_prev = oracle_objective(N, P, K, X, Om, W, H);
    int it = 0;
    if (trace) trace[0] = f_prev;
    while (it < max_iters) {
        oracle_h_step(N, P, K, X, Om, W, H);
        oracle_w_step(N, P, K, X, Om, W, H);
        ++it;
        if (it % check_every == 0) {
            const double f = oracle_objective(N, P, K, X, Om, W, H);
            const int stop = fabs(f_prev - f) < tol * f_prev;
            if (trace) trace[it / check_every] = f;
            f_prev = f;
            if (stop) break;
        }
    }
    if (f_last) *f_last = f_prev;
    return it;
}

/* ---- derotate + stack ------------------------------------------- */
/* the PSF-subtracted images "are rotated North-up using their position angles
 * ... then combined"; PAPER.md:99 likewise for MIRI.  The paper delegates both steps to
 * third-party tools and states no convention.  Readings (G22-G25):
 *  G22  frames are ny x nx images, pixel (y, x) at index y*nx + x, rotation centre at the
 *       pixel (cy, cx) = (ny/2, nx/2) (integer division; the generators' star position).
 *       Frame m is rotated by angle[m] degrees, counter-clockwise with x to the right and
 *       y (row index) up: output pixel (y, x) takes the input at
 *         xs = cx + c*(x-cx) + s*(y-cy),   ys = cy - s*(x-cx) + c*(y-cy),  (s, c) = sin, cos(angle),
 *       evaluated in fp64 with quadrant-exact sine/cosine (multiples of 90 degrees move
 *       pixels exactly).  The caller supplies the rotation to apply (the sign that takes a
 *       position angle to North-up is an instrument convention the paper does not state).
 *  G23  bilinear interpolation over the four neighbours (y0, x0) .. (y0+1, x0+1),
 *       (x0, y0) = floor(xs, ys).  Neighbours with weight <= 1e-6 are ignored.  The
 *       sample is valid only if every remaining neighbour lies inside the image and
 *       (when a weight/mask frame is given) has omega > 0; otherwise frame m contributes
 *       nothing at this pixel ("missing data").  Weights are not renormalised.
 *  G24  combination = mean over the frames with a valid sample (the paper says only
 *       "combined"); a pixel with no valid sample gets `fill`.  count (nullable) receives
 *       the number of frames averaged.
 * Pins: tests/test_oracle_pins.py P20-P24.  Only the interpolation / combination
 * conventions above are "parity unpinned" against the paper (it states none); the
 * arithmetic they define is pinned.                                                         */
static void sincos_deg(double deg, double* s, double* c) {
    double a = fmod(deg, 360.0);
    if (a < 0.0) a += 360.0;
    const int k = (int)floor(a / 90.0 + 0.5);            /* nearest multiple of 90: 0..4 */
    const double r = (a - 90.0 * k) * (3.14159265358979323846 / 180.0);
    const double sr = sin(r), cr = cos(r);               /* |r| <= 45 degrees; r = 0 gives exactly (0, 1) */
    switch (k & 3) {
        case 0: *s = sr;  *c = cr;  break;
        case 1: *s = cr;  *c = -sr; break;
        case 2: *s = -sr; *c = -cr; break;
        default: *s = -cr; *c = sr; break;
    }
}

void oracle_derotate_stack(int M, int ny, int nx, const float* R /* [M, ny*nx] */,
                           const float* om /* [M, ny*nx] nullable */, const double* angle_deg /* [M] */,
                           double fill, double* out /* [ny*nx] */, int* count /* [ny*nx] nullable */) {
    const long P = (long)ny * nx;
    const int cy = ny / 2, cx = nx / 2;
    double* sn = (double*)malloc(sizeof(double) * M);
    double* cs = (double*)malloc(sizeof(double) * M);
    for (int m = 0; m < M; ++m) sincos_deg(angle_deg[m], &sn[m], &cs[m]);
#pragma omp parallel for schedule(static)
    for (int y = 0; y < ny; ++y)
        for (int x = 0; x < nx; ++x) {
            const double dx = x - cx, dy = y - cy;
            double sum = 0.0;
            int cnt = 0;
            for (int m = 0; m < M; ++m) {
                const double xs = cx + cs[m] * dx + sn[m] * dy;
                const double ys = cy - sn[m] * dx + cs[m] * dy;
                const double x0 = floor(xs), y0 = floor(ys);
                const double fx = xs - x0, fy = ys - y0;
                const double w[4] = {(1.0 - fx) * (1.0 - fy), fx * (1.0 - fy), (1.0 - fx) * fy, fx * fy};
                int valid = 1;
                double v = 0.0;
                for (int i = 0; i < 4; ++i) {
                    if (!(w[i] > 1e-6)) continue;
                    const double xi = x0 + (i & 1), yi = y0 + (i >> 1);
                    if (xi < 0 || xi >= nx || yi < 0 || yi >= ny) { valid = 0; break; }
                    const size_t j = (size_t)m * P + (size_t)yi * nx + (size_t)xi;
                    if (om && !((double)om[j] > 0.0)) { valid = 0; break; }
                    v += w[i] * (double)R[j];
                }
                if (valid) { sum += v; ++cnt; }
            }
            out[(size_t)y * nx + x] = cnt ? sum / cnt : fill;
            if (count) count[(size_t)y * nx + x] = cnt;
        }
    free(sn); free(cs);
}
