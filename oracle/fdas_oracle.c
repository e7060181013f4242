/*
 * fdas_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64 (long double where stated) CPU statement of what the FDAS
 * Fourier-domain convolution stage computes.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load this.  It shares no
 * code, header, table or constant generator with the CUDA library under
 * paper_2206_12205_b200/csrc/.
 *
 * What it follows (PAPER.md = /root/reference/PAPER.md, arxiv 2206.12205):
 *   - PAPER.md:35, :49, :59  "convolving the frequency spectrum of the observed time
 *     series with templates"; "The signal is convolved with all templates resulting
 *     in the f-fdot plane"; a pulsar "will appear as a peak on this plane".
 *   - PAPER.md:53-57 (Eq. 1)  z = Fourier bin drift over the observation.
 *   - PAPER.md:65-67  overlap-save computes the SAME windowed convolution with the
 *     contaminated edges discarded, so the plain definition (a direct sum, no FFT,
 *     no segmentation) is the oracle.
 *   - PAPER.md:37, :105  the template is the Fourier response of a constant-fdot
 *     signal (Ransom et al. 2002); the paper does not print it, so it is written
 *     here from the constant-fdot phase model itself (reading A1):
 *         W_z(q) = int_0^1 exp(2 pi i [ q u + (z/2)(u^2 - u) ]) du
 *     = response, q bins away from the MEAN frequency, of a unit complex tone whose
 *     frequency rises by z bins over the observation.  It is evaluated by composite
 *     Gauss-Legendre quadrature of that integral in long double -- i.e. the
 *     definition, not a Fresnel closed form (the closed form lives in
 *     oracle/reference.py and the two are pinned against each other, tests P1).
 *   - template taps h_z[j] = conj(W_z(j)), j = -m_z..m_z, m_z = ceil(|z|/2) + 16
 *     (BASELINE.json configs: "half-width ceil(|z|/2)+16"); zero elsewhere; no
 *     renormalisation (readings A4-A6).
 *   - Y_z[r] = sum_j X[r-j] h_z[j], X = 0 outside [0, M)  (reading A7);
 *     P[z][r] = Re(Y)^2 + Im(Y)^2  (PAPER.md:59 "plane of power", :225).
 *   - peaks: threshold + 8-neighbour local maximum with a lexicographic tie-break
 *     (PAPER.md:186-188 take "the highest point"; reading A14).
 *
 * Parity pins: every function here is pinned by tests/test_oracle_*.py against
 * closed forms / invariants / brute force (P1-P15 in DESIGN.md).  Nothing is
 * "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_GL_NODES 16
#define ORACLE_GL_PANELS 128

static const long double PI_L = 3.14159265358979323846264338327950288L;

/* m_z = ceil(|z|/2) + 16  (BASELINE.json configs). */
int fdas_oracle_halfwidth(double z)
{
    return (int)ceil(fabs(z) / 2.0) + 16;
}

int fdas_oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* n-point Gauss-Legendre nodes x[i] in (-1,1) and weights w[i]; Newton iteration on
 * the Legendre polynomial P_n (textbook: three-term recurrence + derivative). */
static void gauss_legendre(int n, long double *x, long double *w)
{
    for (int i = 0; i < n; ++i) {
        long double t = cosl(PI_L * ((long double)i + 0.75L) / ((long double)n + 0.5L));
        long double dp = 1.0L;
        for (int it = 0; it < 100; ++it) {
            long double p0 = 1.0L, p1 = t;
            for (int k = 2; k <= n; ++k) {
                long double pk = ((2.0L * k - 1.0L) * t * p1 - (k - 1.0L) * p0) / (long double)k;
                p0 = p1;
                p1 = pk;
            }
            dp = (long double)n * (t * p1 - p0) / (t * t - 1.0L);
            long double dt = p1 / dp;
            t -= dt;
            if (fabsl(dt) < 1e-21L) break;
        }
        /* recompute derivative at the converged node */
        {
            long double p0 = 1.0L, p1 = t;
            for (int k = 2; k <= n; ++k) {
                long double pk = ((2.0L * k - 1.0L) * t * p1 - (k - 1.0L) * p0) / (long double)k;
                p0 = p1;
                p1 = pk;
            }
            dp = (long double)n * (t * p1 - p0) / (t * t - 1.0L);
        }
        x[i] = t;
        w[i] = 2.0L / ((1.0L - t * t) * dp * dp);
    }
}

/* W_z(q) = int_0^1 exp(2 pi i [q u + (z/2)(u^2 - u)]) du for REAL q (the tests use
 * fractional q for the sinc pin and the injected-signal closed form). */
void fdas_oracle_response(double z, double q, double *re, double *im)
{
    long double xs[ORACLE_GL_NODES], ws[ORACLE_GL_NODES];
    gauss_legendre(ORACLE_GL_NODES, xs, ws);
    long double sr = 0.0L, si = 0.0L;
    const long double h = 1.0L / ORACLE_GL_PANELS;
    for (int p = 0; p < ORACLE_GL_PANELS; ++p) {
        long double a = p * h;
        for (int i = 0; i < ORACLE_GL_NODES; ++i) {
            long double u = a + 0.5L * h * (xs[i] + 1.0L);
            long double cyc = (long double)q * u + 0.5L * (long double)z * (u * u - u);
            cyc -= floorl(cyc);
            long double wgt = 0.5L * h * ws[i];
            sr += wgt * cosl(2.0L * PI_L * cyc);
            si += wgt * sinl(2.0L * PI_L * cyc);
        }
    }
    *re = (double)sr;
    *im = (double)si;
}

/* taps[2*(j+m)+0/1] = Re/Im h_z[j] = conj(W_z(j)), j = -m..m. */
int fdas_oracle_template(double z, int m, double *taps)
{
    if (m < 0 || !taps) return 1;
    long double xs[ORACLE_GL_NODES], ws[ORACLE_GL_NODES];
    gauss_legendre(ORACLE_GL_NODES, xs, ws);
    const long double h = 1.0L / ORACLE_GL_PANELS;
#pragma omp parallel for schedule(static)
    for (int j = -m; j <= m; ++j) {
        long double sr = 0.0L, si = 0.0L;
        for (int p = 0; p < ORACLE_GL_PANELS; ++p) {
            long double a = p * h;
            for (int i = 0; i < ORACLE_GL_NODES; ++i) {
                long double u = a + 0.5L * h * (xs[i] + 1.0L);
                long double cyc = (long double)j * u + 0.5L * (long double)z * (u * u - u);
                cyc -= floorl(cyc);
                long double wgt = 0.5L * h * ws[i];
                sr += wgt * cosl(2.0L * PI_L * cyc);
                si += wgt * sinl(2.0L * PI_L * cyc);
            }
        }
        taps[2 * (j + m) + 0] = (double)sr;
        taps[2 * (j + m) + 1] = (double)(-si); /* conj */
    }
    return 0;
}

/* Jerk extension (section 2.2: "Jerk Searching takes into account a change in
 * acceleration, and therefore extends the f-fdot plane into an f-fdot-fddot volume ... based on the
 * same principal of convolving templates").  One slab of that volume = one f-fdot plane at a fixed
 * jerk w (change of the drift over the observation, in Fourier bins).  Reading A25: the
 * instantaneous frequency is r0 + z (u - 1/2) + (w/2)(u^2 - u + 1/6), whose mean is r0 and whose
 * mean slope is z, so the response is
 *   W_{z,w}(q) = int_0^1 exp(2 pi i [q u + (z/2)(u^2 - u) + (w/12)(2u^3 - 3u^2 + u)]) du ,
 * taps h_{z,w}[j] = conj(W_{z,w}(j)), |j| <= m = ceil(|z|/2 + |w|/12) + 16 (the largest frequency
 * excursion from the mean is |z|/2 + |w|/12).  w = 0 is the constant-acceleration response. */
int fdas_oracle_halfwidth_jerk(double z, double w)
{
    return (int)ceil(fabs(z) / 2.0 + fabs(w) / 12.0) + 16;
}

void fdas_oracle_response_jerk(double z, double w, double q, double *re, double *im)
{
    long double xs[ORACLE_GL_NODES], ws[ORACLE_GL_NODES];
    gauss_legendre(ORACLE_GL_NODES, xs, ws);
    long double sr = 0.0L, si = 0.0L;
    const long double h = 1.0L / ORACLE_GL_PANELS;
    for (int p = 0; p < ORACLE_GL_PANELS; ++p) {
        long double a = p * h;
        for (int i = 0; i < ORACLE_GL_NODES; ++i) {
            long double u = a + 0.5L * h * (xs[i] + 1.0L);
            long double cyc = (long double)q * u + 0.5L * (long double)z * (u * u - u) +
                              ((long double)w / 12.0L) * (2.0L * u * u * u - 3.0L * u * u + u);
            cyc -= floorl(cyc);
            long double wgt = 0.5L * h * ws[i];
            sr += wgt * cosl(2.0L * PI_L * cyc);
            si += wgt * sinl(2.0L * PI_L * cyc);
        }
    }
    *re = (double)sr;
    *im = (double)si;
}

int fdas_oracle_template_jerk(double z, double w, int m, double *taps)
{
    if (m < 0 || !taps) return 1;
#pragma omp parallel for schedule(static)
    for (int j = -m; j <= m; ++j) {
        double re, im;
        fdas_oracle_response_jerk(z, w, (double)j, &re, &im);
        taps[2 * (j + m) + 0] = re;
        taps[2 * (j + m) + 1] = -im; /* conj */
    }
    return 0;
}

/* One template row, bins r in [r_begin, r_end):
 *   Y[r] = sum_{j=-m}^{m} X[r-j] h[j]   (X = 0 outside [0,M)),  P[r] = |Y[r]|^2.
 * X is interleaved (re, im) fp64, length M complex.  out has r_end - r_begin entries.
 * If y_out != NULL the complex Y is also written (interleaved). */
int fdas_oracle_row(const double *X, int64_t M, const double *taps, int m,
                    int64_t r_begin, int64_t r_end, double *p_out, double *y_out)
{
    if (!X || !taps || !p_out || M < 0 || m < 0 || r_begin > r_end) return 1;
#pragma omp parallel for schedule(static)
    for (int64_t r = r_begin; r < r_end; ++r) {
        double yr = 0.0, yi = 0.0;
        for (int j = -m; j <= m; ++j) {
            int64_t k = r - j;
            if (k < 0 || k >= M) continue;
            double xr = X[2 * k], xi = X[2 * k + 1];
            double hr = taps[2 * (j + m)], hi = taps[2 * (j + m) + 1];
            yr += xr * hr - xi * hi;
            yi += xr * hi + xi * hr;
        }
        p_out[r - r_begin] = yr * yr + yi * yi;
        if (y_out) {
            y_out[2 * (r - r_begin)] = yr;
            y_out[2 * (r - r_begin) + 1] = yi;
        }
    }
    return 0;
}

/* Whole plane (or a column window of it): templates z_k = -zmax + k*dz, k = 0..K-1,
 * K = 2*floor(zmax/dz) + 1; plane[k*(r_end-r_begin) + (r - r_begin)]. */
int fdas_oracle_plane(const double *X, int64_t M, double zmax, double dz,
                      int64_t r_begin, int64_t r_end, double *plane)
{
    if (!X || !plane || dz <= 0.0 || zmax < 0.0 || r_begin < 0 || r_end > M || r_begin > r_end)
        return 1;
    int K = 2 * (int)floor(zmax / dz + 1e-9) + 1;
    int64_t W = r_end - r_begin;
    for (int k = 0; k < K; ++k) {
        double z = -zmax + k * dz;
        int m = fdas_oracle_halfwidth(z);
        double *taps = (double *)malloc(sizeof(double) * 2 * (2 * m + 1));
        if (!taps) return 2;
        fdas_oracle_template(z, m, taps);
        fdas_oracle_row(X, M, taps, m, r_begin, r_end, plane + (int64_t)k * W, NULL);
        free(taps);
    }
    return 0;
}

/* Peaks (reading A14): (k, r) is a peak iff P > thr and P >= every existing
 * 8-neighbour, strictly > for neighbours that precede (k, r) in (k, r) lexicographic
 * order (a plateau gives exactly one peak: its lexicographically first cell).  out[3*i] = k, r, power; returns the TOTAL count; only the first
 * `capacity` (in row-major scan order) are written. */
int64_t fdas_oracle_peaks(const double *P, int K, int64_t M, double thr,
                          double *out, int64_t capacity)
{
    int64_t count = 0;
    for (int k = 0; k < K; ++k) {
        for (int64_t r = 0; r < M; ++r) {
            double v = P[(int64_t)k * M + r];
            if (!(v > thr)) continue;
            int ok = 1;
            for (int dk = -1; dk <= 1 && ok; ++dk) {
                for (int dr = -1; dr <= 1; ++dr) {
                    if (dk == 0 && dr == 0) continue;
                    int kk = k + dk;
                    int64_t rr = r + dr;
                    if (kk < 0 || kk >= K || rr < 0 || rr >= M) continue;
                    double n = P[(int64_t)kk * M + rr];
                    int precedes = (dk < 0) || (dk == 0 && dr < 0);
                    if (precedes ? !(v > n) : !(v >= n)) { ok = 0; break; }
                }
            }
            if (ok) {
                if (count < capacity && out) {
                    out[3 * count + 0] = (double)k;
                    out[3 * count + 1] = (double)r;
                    out[3 * count + 2] = v;
                }
                ++count;
            }
        }
    }
    return count;
}

/* Peaks of an f-fdot-fddot volume (the jerk search "extends the f-fdot plane into an
 * f-fdot-fddot volume"; reading A27): V[i][k][r], i = 0..W-1 the jerk slab, k the template row, r the
 * bin.  The plane rule (reading A14) with one more axis: (i, k, r) is a peak iff V > thr and V >= every existing
 * one of its 26 neighbours, strictly > for neighbours that precede it in (i, k, r) lexicographic order (a
 * plateau gives exactly one peak).  out[4*n] = i, k, r, power; returns the TOTAL count; only the first
 * `capacity` (in scan order) are written.  W = 1 is fdas_oracle_peaks. */
int64_t fdas_oracle_peaks3(const double *V, int W, int K, int64_t M, double thr, double *out, int64_t capacity)
{
    int64_t count = 0;
    for (int i = 0; i < W; ++i) {
        for (int k = 0; k < K; ++k) {
            for (int64_t r = 0; r < M; ++r) {
                double v = V[((int64_t)i * K + k) * M + r];
                if (!(v > thr)) continue;
                int ok = 1;
                for (int di = -1; di <= 1 && ok; ++di) {
                    for (int dk = -1; dk <= 1 && ok; ++dk) {
                        for (int dr = -1; dr <= 1; ++dr) {
                            if (di == 0 && dk == 0 && dr == 0) continue;
                            int ii = i + di, kk = k + dk;
                            int64_t rr = r + dr;
                            if (ii < 0 || ii >= W || kk < 0 || kk >= K || rr < 0 || rr >= M) continue;
                            double n = V[((int64_t)ii * K + kk) * M + rr];
                            int precedes = (di < 0) || (di == 0 && (dk < 0 || (dk == 0 && dr < 0)));
                            if (precedes ? !(v > n) : !(v >= n)) { ok = 0; break; }
                        }
                    }
                }
                if (ok) {
                    if (count < capacity && out) {
                        out[4 * count + 0] = (double)i;
                        out[4 * count + 1] = (double)k;
                        out[4 * count + 2] = (double)r;
                        out[4 * count + 3] = v;
                    }
                    ++count;
                }
            }
        }
    }
    return count;
}
