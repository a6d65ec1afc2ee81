/*
 * tina_oracle.c -- float64 CPU oracle for the FIR / DFT / IDFT / PFB path of
 * arxiv 2408.16551 (TINA).  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  It shares no code,
 * table, header or helper with the CUDA path under paper_2408_16551_b200/.
 *
 * Every function is the plain definition of the result, written as plain
 * loops in the paper's index order, in double precision:
 *
 *   oracle_fir   Eq. (15), PAPER.md:171      y(i) = sum_k a(k) x(i-k)
 *   oracle_dft   Eq. (12)/(14), PAPER.md:146/:158   Z = X.F , X = Z.IF
 *   oracle_pfb   Eq. (20), followed by the DFT of sec. 4.1
 *
 *   oracle_unfold Eq. (17), PAPER.md:187     Y(i,j) = X(i+j)
 *   oracle_mul / oracle_add / oracle_sum / oracle_matmul   Eq. (6), (10), (11), (7): PAPER.md:96, :127,
 *                :136, :104 -- the arithmetic building blocks of section 3
 *
 * Readings of the paper where it is silent (SURVEY.md
 * section 8(c) R1..R16): 0-based sums, valid mode, x_p(n') = x[n'P+p],
 * h_p(m) = w[mP+p], forward DFT unnormalised with exp(-2 pi i ln/N), inverse
 * with exp(+...) and 1/N.
 *
 * Pins: tests/test_oracle_pins.py (none of them re-types these formulas).
 * OpenMP is used only over the outermost independent index; no sum changes
 * its order.
 */
#include <math.h>
#include <stddef.h>
#include <stdlib.h>

#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_PI 3.14159265358979323846264338327950288

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* Eq. (15), valid mode (reading R3):
 *   y[c][j] = sum_{k=0}^{K-1} a[k] * x[c][j + K-1 - k],  j in [0, L-K+1).
 * With i = j + K-1 this is y(i) = sum_k a(k) x(i-k) for every i whose whole
 * history x(i-K+1..i) exists.  One tap vector for all C channels (R13).
 * x: [C][L] float32, a: [K] float32, y: [C][L-K+1] float64.                 */
int oracle_fir(const float *x, const float *a, double *y,
               long long C, long long L, long long K)
{
    if (!x || !a || !y || C < 1 || K < 1 || L < K) return 1;
    const long long Lo = L - K + 1;
    long long c;
#pragma omp parallel for schedule(static)
    for (c = 0; c < C; ++c) {
        for (long long j = 0; j < Lo; ++j) {
            double acc = 0.0;
            for (long long k = 0; k < K; ++k)
                acc += (double)a[k] * (double)x[c * L + (j + K - 1 - k)];
            y[c * Lo + j] = acc;
        }
    }
    return 0;
}

/* Eq. (15), with one tap vector PER CHANNEL -- the "multiple FIR filters"
 * that the PFB's subfilter stage combines (Eq. (20): branch p is
 * filtered with its own h_p).  Valid mode as above:
 *   y[c][j] = sum_{k=0}^{K-1} a[c][k] * x[c][j + K-1 - k],  j in [0, L-K+1).
 * x: [C][L] float32, a: [C][K] float32, y: [C][L-K+1] float64.              */
int oracle_fir_multi(const float *x, const float *a, double *y,
                     long long C, long long L, long long K)
{
    if (!x || !a || !y || C < 1 || K < 1 || L < K) return 1;
    const long long Lo = L - K + 1;
    long long c;
#pragma omp parallel for schedule(static)
    for (c = 0; c < C; ++c) {
        for (long long j = 0; j < Lo; ++j) {
            double acc = 0.0;
            for (long long k = 0; k < K; ++k)
                acc += (double)a[c * K + k] * (double)x[c * L + (j + K - 1 - k)];
            y[c * Lo + j] = acc;
        }
    }
    return 0;
}

/* Eq. (17): Y(i,j) = X(i+j), output (I-J+1) x J.               */
int oracle_unfold(const float *x, double *y, long long I, long long J)
{
    if (!x || !y || J < 1 || I < J) return 1;
    for (long long i = 0; i < I - J + 1; ++i)
        for (long long j = 0; j < J; ++j)
            y[i * J + j] = (double)x[i + j];
    return 0;
}

/* Eq. (6): O(c) = I(c) K(c).                                     */
int oracle_mul(const float *a, const float *b, double *o, long long n)
{
    if (!a || !b || !o || n < 0) return 1;
    for (long long c = 0; c < n; ++c) o[c] = (double)a[c] * (double)b[c];
    return 0;
}

/* Eq. (10): O(c) = b(c) + I(c).                                 */
int oracle_add(const float *a, const float *b, double *o, long long n)
{
    if (!a || !b || !o || n < 0) return 1;
    for (long long c = 0; c < n; ++c) o[c] = (double)b[c] + (double)a[c];
    return 0;
}

/* Eq. (11): O = sum_c I(c), one sum per row of x[rows][n], in
 * index order (double accumulation; compensated, so the order does not show). */
int oracle_sum(const float *x, double *o, long long rows, long long n)
{
    if (!x || !o || rows < 0 || n < 0) return 1;
    for (long long r = 0; r < rows; ++r) {
        double acc = 0.0, comp = 0.0;                    /* Neumaier: exact to ~1 ulp of double */
        for (long long c = 0; c < n; ++c) {
            const double v = (double)x[r * n + c], t = acc + v;
            comp += fabs(acc) >= fabs(v) ? (acc - t) + v : (v - t) + acc;
            acc = t;
        }
        o[r] = acc + comp;
    }
    return 0;
}

/* Eq. (7): Z(m,n) = sum_l X(m,l) Y(l,n); X [M][L], Y [L][N],
 * Z [M][N], row-major.                                                        */
int oracle_matmul(const float *x, const float *y, double *z, long long M, long long L, long long N)
{
    if (!x || !y || !z || M < 0 || L < 0 || N < 0) return 1;
#pragma omp parallel for schedule(static)
    for (long long m = 0; m < M; ++m)
        for (long long n = 0; n < N; ++n) {
            double acc = 0.0;
            for (long long l = 0; l < L; ++l) acc += (double)x[m * L + l] * (double)y[l * N + n];
            z[m * N + n] = acc;
        }
    return 0;
}

/* Twiddle table W[r] = exp(sign * 2 pi i r / N), r in [0,N).  The index
 * (n*k) mod N is formed in integers so no large-argument trig is evaluated. */
static int make_table(long long N, int sign, double **wr, double **wi)
{
    *wr = (double *)malloc((size_t)N * sizeof(double));
    *wi = (double *)malloc((size_t)N * sizeof(double));
    if (!*wr || !*wi) { free(*wr); free(*wi); return 1; }
    for (long long r = 0; r < N; ++r) {
        const double th = 2.0 * ORACLE_PI * (double)r / (double)N;
        (*wr)[r] = cos(th);
        (*wi)[r] = (double)sign * sin(th);
    }
    return 0;
}

/* Eq. (12) PAPER.md:146 (forward) and Eq. (14) PAPER.md:158 (inverse):
 *   Z[b][k] = s * sum_{n=0}^{N-1} x[b][n] * exp(-/+ 2 pi i n k / N),
 * s = 1 forward, 1/N inverse (reading R7).
 * x: [B][N] complex64 interleaved (re,im float32); z: [B][N] complex128
 * interleaved.                                                               */
int oracle_dft(const float *x, double *z, long long B, long long N, int inverse)
{
    if (!x || !z || B < 1 || N < 1) return 1;
    double *wr, *wi;
    if (make_table(N, inverse ? +1 : -1, &wr, &wi)) return 2;
    const double s = inverse ? 1.0 / (double)N : 1.0;
    long long b;
#pragma omp parallel for schedule(static)
    for (b = 0; b < B; ++b) {
        const float *xb = x + 2 * b * N;
        for (long long k = 0; k < N; ++k) {
            double ar = 0.0, ai = 0.0;
            for (long long n = 0; n < N; ++n) {
                const long long r = (n * k) % N;
                const double xr = (double)xb[2 * n], xi = (double)xb[2 * n + 1];
                ar += xr * wr[r] - xi * wi[r];
                ai += xr * wi[r] + xi * wr[r];
            }
            z[2 * (b * N + k)]     = s * ar;
            z[2 * (b * N + k) + 1] = s * ai;
        }
    }
    free(wr); free(wi);
    return 0;
}

/* Same transform on float64 input (used by pins that chain IDFT(DFT(x))
 * without an intermediate rounding to float32).                              */
int oracle_dft_f64(const double *x, double *z, long long B, long long N, int inverse)
{
    if (!x || !z || B < 1 || N < 1) return 1;
    double *wr, *wi;
    if (make_table(N, inverse ? +1 : -1, &wr, &wi)) return 2;
    const double s = inverse ? 1.0 / (double)N : 1.0;
    long long b;
#pragma omp parallel for schedule(static)
    for (b = 0; b < B; ++b) {
        const double *xb = x + 2 * b * N;
        for (long long k = 0; k < N; ++k) {
            double ar = 0.0, ai = 0.0;
            for (long long n = 0; n < N; ++n) {
                const long long r = (n * k) % N;
                ar += xb[2 * n] * wr[r] - xb[2 * n + 1] * wi[r];
                ai += xb[2 * n] * wi[r] + xb[2 * n + 1] * wr[r];
            }
            z[2 * (b * N + k)]     = s * ar;
            z[2 * (b * N + k) + 1] = s * ai;
        }
    }
    free(wr); free(wi);
    return 0;
}

/* Number of output frames: F = floor(n_samples / P) - M + 1 (readings R3, R8). */
long long oracle_pfb_num_frames(long long n_samples, long long P, long long M)
{
    if (P < 1 || M < 1 || n_samples < 0) return 0;
    return n_samples / P - M + 1;
}

/* Eq. (20) PAPER.md:230 then the DFT of sec. 4.1 across the P branches
 * (PAPER.md:233), for the frames listed in frames[0..n_sel) (frames == NULL
 * means all frames 0..F-1 in order):
 *   y[f][p] = sum_{m=0}^{M-1} w[m P + p] * x[(f + M-1 - m) P + p]
 *   X[f][k] = sum_{p=0}^{P-1} y[f][p] * exp(-2 pi i ((p k) mod P) / P)
 * i.e. x_p(n') = x[n' P + p], h_p(m) = w[m P + p], frame f <-> n' = f + M-1
 * (readings R4, R5, R6).  is_real = 0: x is complex64 interleaved, k in
 * [0,P); is_real = 1: x is float32, k in [0, P/2] (reading R12).
 * out_y (optional, may be NULL): [n_sel][P] complex128 (or float64 if real)
 * subfiltered signals; out_X: [n_sel][NK] complex128 interleaved.            */
int oracle_pfb(const float *x, long long n_samples, long long P, long long M,
               const float *w, int is_real,
               const long long *frames, long long n_sel,
               double *out_y, double *out_X)
{
    if (!x || !w || !out_X || P < 1 || M < 1) return 1;
    if (is_real && (P % 2)) return 1;
    const long long F = oracle_pfb_num_frames(n_samples, P, M);
    if (F < 1) return 1;
    if (!frames) n_sel = F;
    const long long NK = is_real ? P / 2 + 1 : P;
    double *wr, *wi;
    if (make_table(P, -1, &wr, &wi)) return 2;
    int bad = 0;
    long long s;
#pragma omp parallel for schedule(dynamic, 1)
    for (s = 0; s < n_sel; ++s) {
        const long long f = frames ? frames[s] : s;
        if (f < 0 || f >= F) { bad = 1; continue; }
        double *yr = (double *)malloc((size_t)P * sizeof(double));
        double *yi = (double *)malloc((size_t)P * sizeof(double));
        for (long long p = 0; p < P; ++p) {
            double ar = 0.0, ai = 0.0;
            for (long long m = 0; m < M; ++m) {
                const double h = (double)w[m * P + p];
                const long long n = (f + M - 1 - m) * P + p;
                if (is_real) {
                    ar += h * (double)x[n];
                } else {
                    ar += h * (double)x[2 * n];
                    ai += h * (double)x[2 * n + 1];
                }
            }
            yr[p] = ar; yi[p] = ai;
            if (out_y) {
                if (is_real) out_y[s * P + p] = ar;
                else { out_y[2 * (s * P + p)] = ar; out_y[2 * (s * P + p) + 1] = ai; }
            }
        }
        for (long long k = 0; k < NK; ++k) {
            double ar = 0.0, ai = 0.0;
            for (long long p = 0; p < P; ++p) {
                const long long r = (p * k) % P;
                ar += yr[p] * wr[r] - yi[p] * wi[r];
                ai += yr[p] * wi[r] + yi[p] * wr[r];
            }
            out_X[2 * (s * NK + k)]     = ar;
            out_X[2 * (s * NK + k) + 1] = ai;
        }
        free(yr); free(yi);
    }
    free(wr); free(wi);
    return bad;
}
