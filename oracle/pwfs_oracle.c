/*
 * pwfs_oracle.c -- ORACLE (test infrastructure, NOT the product).
 *
 * Plain, slow, double-precision CPU statement of the modulated pyramid
 * wavefront-sensor forward model.  It exists only so that tests/, the smoke
 * check in __graft_entry__.py and bench.py's cpu_baseline / --impl reference
 * legs have something independent to compare the CUDA path with.  The product
 * path (paper_1607_07624_b200/) never imports, links or executes this file,
 * and this file shares no code, header, table or constant with the CUDA path.
 *
 * What it follows.  The paper only names the object: "apply a
 * transformation from focal plane to pupil plane emulating an optical
 * pyramid" (section 2), parameters at PAPER.md:L119-136
 * (Table 1, `pyramid`), data flow pyr.in_ef -> pyr.out_i -> ccd.in_i ->
 * ccd.out_pixels -> sc.in_pixels -> sc.out_slopes (PAPER.md:L261-262,
 * L317-318), and lists it as GPU-accelerated "Pyramid ... propagation (from
 * wavefront to detector plane)" (section 6).  The arithmetic
 * is the step list of BASELINE.json `north_star`, written out as definitions
 * O0..O9 in SURVEY.md section 8(c); each function below cites its O-number.
 * Every reading of a silent point (A1..A16 of SURVEY.md 8(c)) is repeated in
 * DESIGN.md.
 *
 * The FFT reaches exactly (up to rounding order) the DFT's result, so the
 * reference definition is orc_dft_naive(); orc_fft() is a textbook recursive
 * mixed-radix Cooley-Tukey used only for speed and is pinned to the naive DFT
 * and to numpy.fft in tests/test_oracle_fft.py.
 *
 * Pins (tests/, -m "not gpu"): brute-force DFT, Parseval, flat-phase mirror
 * symmetry and zero slopes, +-tilt antisymmetry, small-tilt linearity,
 * identity mask, single-face ramp == circular shift, integer-bin tilt ==
 * circular shift of F, geometric-optics gain (2/pi)asin(alpha/r), separable
 * circulant operator on tiny grids, rebin partition of unity, valid-mask
 * counts.  Nothing the paper prints can be compared (it prints no number for
 * this path): parity WITH THE PAPER is unpinned; parity with the mathematics
 * is pinned by the list above.
 *
 * Conventions: arrays are row-major [y][x] (x fast).  `sign` = -1 forward,
 * +1 inverse; transforms here are UNNORMALISED unless stated.
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex zc;

#define ORC_OK 0
#define ORC_EINVAL (-1)
#define ORC_ENOMEM (-2)

static const double TWO_PI = 6.283185307179586476925286766559;

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---------------------------------------------------------------- DFT ---- */

/* Definition of the DFT:  out[k] = sum_j in[j] exp(sign 2 pi i j k / n).
 * (north_star: "naive DFT"; SURVEY 8(c) O3/O5 in one dimension.) */
void orc_dft_naive(int n, const zc *in, zc *out, int sign) {
    for (int k = 0; k < n; ++k) {
        zc acc = 0.0;
        for (int j = 0; j < n; ++j) {
            /* reduce j*k mod n in integers so the angle stays accurate */
            long long jk = ((long long)j * k) % n;
            double ang = sign * TWO_PI * (double)jk / (double)n;
            acc += in[j] * (cos(ang) + I * sin(ang));
        }
        out[k] = acc;
    }
}

static int smallest_factor(int n) {
    for (int p = 2; (long long)p * p <= n; ++p)
        if (n % p == 0) return p;
    return n;
}

/* Textbook recursive decimation-in-time Cooley-Tukey for n = p*q:
 *   Y_r[k]      = DFT_q( in[r + p j] )_k                 r = 0..p-1
 *   out[k + q t] = sum_r w_n^{r (k + q t)} Y_r[k]         t = 0..p-1
 * with w_n = exp(sign 2 pi i / n) read from a table `w` of the TOP-level size
 * n_top (w[m] = exp(sign 2 pi i m / n_top)); prime n falls back to the
 * definition.  No blocking, no reordering beyond the recursion itself. */
static void fft_rec(int n, int stride, const zc *in, zc *out, const zc *w,
                    int n_top, zc *scratch) {
    if (n == 1) { out[0] = in[0]; return; }
    int p = smallest_factor(n);
    int step = n_top / n;                      /* w_n^m = w[(m mod n) * step] */
    if (p == n) {                              /* prime length: definition */
        for (int k = 0; k < n; ++k) {
            zc acc = 0.0;
            for (int j = 0; j < n; ++j)
                acc += in[(size_t)j * stride] * w[(size_t)(((long long)j * k) % n) * step];
            out[k] = acc;
        }
        return;
    }
    int q = n / p;
    zc *Y = scratch;                           /* p*q values */
    for (int r = 0; r < p; ++r)
        fft_rec(q, stride * p, in + (size_t)r * stride, Y + (size_t)r * q, w, n_top,
                scratch + n);
    for (int k = 0; k < q; ++k)
        for (int t = 0; t < p; ++t) {
            int ko = k + q * t;
            zc acc = 0.0;
            for (int r = 0; r < p; ++r)
                acc += Y[(size_t)r * q + k] * w[(size_t)(((long long)r * ko) % n) * step];
            out[ko] = acc;
        }
}

static zc *make_twiddles(int n, int sign) {
    zc *w = (zc *)malloc(sizeof(zc) * (size_t)n);
    if (!w) return NULL;
    for (int m = 0; m < n; ++m) {
        double ang = sign * TWO_PI * (double)m / (double)n;
        w[m] = cos(ang) + I * sin(ang);
    }
    return w;
}

/* 1-D FFT, any n >= 1 (fast for 2/3/5-smooth n).  in != out. */
int orc_fft(int n, const zc *in, zc *out, int sign) {
    if (n < 1 || (sign != 1 && sign != -1)) return ORC_EINVAL;
    zc *w = make_twiddles(n, sign);
    zc *scratch = (zc *)malloc(sizeof(zc) * (size_t)(2 * n + 64));
    if (!w || !scratch) { free(w); free(scratch); return ORC_ENOMEM; }
    fft_rec(n, 1, in, out, w, n, scratch);
    free(w); free(scratch);
    return ORC_OK;
}

/* 2-D transform of an M x M array, in place:
 *   a[v][u] <- sum_y sum_x a[y][x] exp(sign 2 pi i (u x + v y)/M)
 * done as M row transforms followed by M column transforms (the 2-D DFT is
 * separable).  use_naive != 0 uses the O(M^2) definition for each 1-D pass. */
int orc_fft2(int M, zc *a, int sign, int use_naive) {
    if (M < 1) return ORC_EINVAL;
    zc *w = make_twiddles(M, sign);
    zc *line = (zc *)malloc(sizeof(zc) * (size_t)M);
    zc *res = (zc *)malloc(sizeof(zc) * (size_t)M);
    zc *scratch = (zc *)malloc(sizeof(zc) * (size_t)(2 * M + 64));
    if (!w || !line || !res || !scratch) { free(w); free(line); free(res); free(scratch); return ORC_ENOMEM; }
    for (int y = 0; y < M; ++y) {              /* rows: x -> u */
        memcpy(line, a + (size_t)y * M, sizeof(zc) * (size_t)M);
        if (use_naive) orc_dft_naive(M, line, res, sign);
        else fft_rec(M, 1, line, res, w, M, scratch);
        memcpy(a + (size_t)y * M, res, sizeof(zc) * (size_t)M);
    }
    for (int u = 0; u < M; ++u) {              /* columns: y -> v */
        for (int y = 0; y < M; ++y) line[y] = a[(size_t)y * M + u];
        if (use_naive) orc_dft_naive(M, line, res, sign);
        else fft_rec(M, 1, line, res, w, M, scratch);
        for (int v = 0; v < M; ++v) a[(size_t)v * M + u] = res[v];
    }
    free(w); free(line); free(res); free(scratch);
    return ORC_OK;
}

/* ------------------------------------------------ O0..O6: the optics ---- */

/* O0: modulation points on the circle.  theta_k = theta0 + 2 pi k / K,
 * (dx_k, dy_k) = r (cos theta_k, sin theta_k) in lambda/D (reading A4:
 * start on +x, counter-clockwise, equally spaced). */
void orc_mod_offsets(int K, double r, double theta0, double *dx, double *dy) {
    for (int k = 0; k < K; ++k) {
        double th = theta0 + TWO_PI * (double)k / (double)K;
        dx[k] = r * cos(th);
        dy[k] = r * sin(th);
    }
}

/* O1: pupil phasor with the modulation tilt,
 *   P[y][x] = A[y][x] exp(i (phi[y][x] + 2 pi (dx (x-c) + dy (y-c)) / N)),
 * c = (N-1)/2.  (north_star: "builds the pupil phasor A exp(i(phi+tilt_k))";
 * readings A1-A3: phi in radians, D spans N px so 1 lambda/D = 2 pi over N px,
 * tilt about the pupil centre.)  A, phi are float32 and are widened exactly. */
void orc_phasor(int N, const float *A, const float *phi, double dx, double dy, zc *P) {
    double c = 0.5 * (double)(N - 1);
    for (int y = 0; y < N; ++y)
        for (int x = 0; x < N; ++x) {
            double tilt = TWO_PI * (dx * ((double)x - c) + dy * ((double)y - c)) / (double)N;
            double ph = (double)phi[(size_t)y * N + x] + tilt;
            P[(size_t)y * N + x] = (double)A[(size_t)y * N + x] * (cos(ph) + I * sin(ph));
        }
}

/* O2: zero-pad into the M x M grid, pupil centred: offset o = M/2 - N/2 on
 * both axes (reading A6). */
void orc_embed(int N, int M, const zc *P, zc *G) {
    int o = M / 2 - N / 2;
    memset(G, 0, sizeof(zc) * (size_t)M * M);
    for (int y = 0; y < N; ++y)
        for (int x = 0; x < N; ++x)
            G[(size_t)(y + o) * M + (x + o)] = P[(size_t)y * N + x];
}

/* O4: four-face pyramid phase mask,
 *   m[v][u] = exp(2 pi i s (|u~| + |v~|) / M),   u~ = u (u < M/2) else u - M
 * (BASELINE.json configs[0]: "Pyramid mask phase 2 pi (|fx|+|fy|) M/4 in
 * cycles/px, placing the four pupil images at +-M/4 offsets"; reading A8:
 * signed frequency in [-M/2, M/2), sign +, ideal edges, no field stop). */
void orc_pyramid_mask(int M, double s, zc *m) {
    for (int v = 0; v < M; ++v) {
        int vs = (v < M / 2) ? v : v - M;
        for (int u = 0; u < M; ++u) {
            int us = (u < M / 2) ? u : u - M;
            double ang = TWO_PI * s * (double)(abs(us) + abs(vs)) / (double)M;
            m[(size_t)v * M + u] = cos(ang) + I * sin(ang);
        }
    }
}

/* O3 + O4 + O5 for one modulation point: E = IDFT2( DFT2(G) * m ) / M^2.
 * F (optional, may be NULL) receives the unnormalised focal-plane field O3.
 * (north_star: "applies a 2D FFT to the focal plane, multiplies by the 4-face
 * pyramid phase mask, applies an inverse 2D FFT back to the pupil plane";
 * reading A7: forward sign -, unnormalised; inverse sign +, 1/M^2.) */
int orc_field(int N, int M, const float *A, const float *phi, double dx, double dy,
              const zc *mask, zc *E, zc *F, int use_naive) {
    if (N < 1 || M < N) return ORC_EINVAL;
    zc *P = (zc *)malloc(sizeof(zc) * (size_t)N * N);
    if (!P) return ORC_ENOMEM;
    orc_phasor(N, A, phi, dx, dy, P);                    /* O1 */
    orc_embed(N, M, P, E);                               /* O2 */
    free(P);
    int rc = orc_fft2(M, E, -1, use_naive);              /* O3 */
    if (rc) return rc;
    if (F) memcpy(F, E, sizeof(zc) * (size_t)M * M);
    for (size_t i = 0; i < (size_t)M * M; ++i) E[i] *= mask[i];   /* O4 */
    rc = orc_fft2(M, E, +1, use_naive);                  /* O5 */
    if (rc) return rc;
    double inv = 1.0 / ((double)M * (double)M);
    for (size_t i = 0; i < (size_t)M * M; ++i) E[i] *= inv;
    return ORC_OK;
}

/* O6: I = (1/K) sum_k |E_k|^2 on the full M x M grid (reading A5: uniform
 * weights, mean).  The k loop is shared among threads; each thread sums its
 * own k's and the per-thread sums are added in thread order. */
int orc_intensity(int N, int M, const float *A, const float *phi, int K, double r,
                  double theta0, const zc *mask, double *Iout, int use_naive) {
    if (K < 1 || N < 1 || M < N) return ORC_EINVAL;
    double *dx = (double *)malloc(sizeof(double) * (size_t)K);
    double *dy = (double *)malloc(sizeof(double) * (size_t)K);
    if (!dx || !dy) { free(dx); free(dy); return ORC_ENOMEM; }
    orc_mod_offsets(K, r, theta0, dx, dy);               /* O0 */
    size_t MM = (size_t)M * M;
    int nt = orc_num_threads();
    if (nt > K) nt = K;
    double *part = (double *)calloc((size_t)nt * MM, sizeof(double));
    int err = part ? ORC_OK : ORC_ENOMEM;
    if (!err) {
#pragma omp parallel num_threads(nt)
        {
#ifdef _OPENMP
            int tid = omp_get_thread_num();
#else
            int tid = 0;
#endif
            zc *E = (zc *)malloc(sizeof(zc) * MM);
            double *acc = part + (size_t)tid * MM;
            if (!E) {
#pragma omp atomic write
                err = ORC_ENOMEM;
            } else {
#pragma omp for schedule(static)
                for (int k = 0; k < K; ++k) {
                    int rc = orc_field(N, M, A, phi, dx[k], dy[k], mask, E, NULL, use_naive);
                    if (rc) {
#pragma omp atomic write
                        err = rc;
                    } else {
                        for (size_t i = 0; i < MM; ++i) {
                            double re = creal(E[i]), im = cimag(E[i]);
                            acc[i] += re * re + im * im;
                        }
                    }
                }
            }
            free(E);
        }
        for (size_t i = 0; i < MM; ++i) {
            double s = 0.0;
            for (int t = 0; t < nt; ++t) s += part[(size_t)t * MM + i];
            Iout[i] = s / (double)K;
        }
    }
    free(part); free(dx); free(dy);
    return err;
}

/* ---------------------------------------- f3: tilt list and field stop ---- */

/* Focal-plane field stop (Table 1
 * `pyramid`: "Requested field-of-view [arcsec]", key lost in extraction).
 * Reading F3a: the stop is the SQUARE |u~| <= h and |v~| <= h in
 * focal-plane bins (signed frequencies as in O4), transmission 1 inside and 0
 * outside, multiplied into the pyramid mask:  m[v][u] <- m[v][u] * stop.
 * h < 0 means "no stop" (mask untouched). */
void orc_field_stop(int M, double h, zc *m) {
    if (h < 0.0) return;
    for (int v = 0; v < M; ++v) {
        int vs = (v < M / 2) ? v : v - M;
        for (int u = 0; u < M; ++u) {
            int us = (u < M / 2) ? u : u - M;
            if ((double)abs(us) > h || (double)abs(vs) > h) m[(size_t)v * M + u] = 0.0;
        }
    }
}

/* O6 generalised to an arbitrary list of tilts with weights (SURVEY.md 8(f)
 * row f3: "replace the K-point circle by an arbitrary list (dx,dy,w) -- covers
 * extended/resolved sources"; "resolved sources", L77):
 *   I = sum_k w_k |E_k|^2 / sum_k w_k,   E_k from O1..O5 with tilt (dx_k, dy_k).
 * Reading F3b: weights are non-negative and normalised by their sum, so the
 * uniform circle list reproduces O6 exactly.  Sequential over k (no threads:
 * this entry is for small pins and parity samples). */
int orc_intensity_list(int N, int M, const float *A, const float *phi, int n_pts,
                       const double *dx, const double *dy, const double *w, const zc *mask,
                       double *Iout, int use_naive) {
    if (n_pts < 1 || N < 1 || M < N) return ORC_EINVAL;
    size_t MM = (size_t)M * M;
    double wsum = 0.0;
    for (int k = 0; k < n_pts; ++k) {
        if (!(w[k] >= 0.0)) return ORC_EINVAL;
        wsum += w[k];
    }
    if (!(wsum > 0.0)) return ORC_EINVAL;
    zc *E = (zc *)malloc(sizeof(zc) * MM);
    if (!E) return ORC_ENOMEM;
    for (size_t i = 0; i < MM; ++i) Iout[i] = 0.0;
    int rc = ORC_OK;
    for (int k = 0; k < n_pts && !rc; ++k) {
        rc = orc_field(N, M, A, phi, dx[k], dy[k], mask, E, NULL, use_naive);
        if (!rc)
            for (size_t i = 0; i < MM; ++i) {
                double re = creal(E[i]), im = cimag(E[i]);
                Iout[i] += w[k] * (re * re + im * im);
            }
    }
    if (!rc)
        for (size_t i = 0; i < MM; ++i) Iout[i] /= wsum;
    free(E);
    return rc;
}

/* ------------------------------------------- O7..O9: detector, slopes ---- */

/* O7 weights: W[i][p] = | [p, p+1) intersect [i b, (i+1) b) |, b = N/n_sub,
 * evaluated in integers scaled by n_sub and divided once (reading A10:
 * n_sub is authoritative, b need not be an integer).  W is n_sub x N. */
void orc_rebin_weights(int N, int n_sub, double *W) {
    for (int i = 0; i < n_sub; ++i)
        for (int p = 0; p < N; ++p) {
            long long lo_pix = (long long)p * n_sub, hi_pix = (long long)(p + 1) * n_sub;
            long long lo_bin = (long long)i * N, hi_bin = (long long)(i + 1) * N;
            long long lo = lo_pix > lo_bin ? lo_pix : lo_bin;
            long long hi = hi_pix < hi_bin ? hi_pix : hi_bin;
            W[(size_t)i * N + p] = (hi > lo) ? (double)(hi - lo) / (double)n_sub : 0.0;
        }
}

/* O7: the four N x N windows of I centred at M/2 +- s are area-weighted-SUMMED
 * into four n_sub x n_sub tiles:
 *   frame[qy n_sub + j][qx n_sub + i] = sum_py sum_px W[j][py] W[i][px]
 *                                       I[wy + py][wx + px],
 *   wx = M/2 + (2 qx - 1) s - N/2 (wy likewise).   frame is 2n_sub x 2n_sub.
 * (north_star: "the summed intensity is then rebinned to the detector's
 * subaperture pixels"; PAPER.md:L318 ccd.in_i = pyr.out_i, noiseless CCD.) */
int orc_frame(int N, int M, int s, int n_sub, const double *Iin, double *frame) {
    if (n_sub < 1 || n_sub > N) return ORC_EINVAL;
    int D = 2 * n_sub;
    double *W = (double *)malloc(sizeof(double) * (size_t)n_sub * N);
    if (!W) return ORC_ENOMEM;
    orc_rebin_weights(N, n_sub, W);
    for (int qy = 0; qy < 2; ++qy)
        for (int qx = 0; qx < 2; ++qx) {
            int wx = M / 2 + (2 * qx - 1) * s - N / 2;
            int wy = M / 2 + (2 * qy - 1) * s - N / 2;
            if (wx < 0 || wy < 0 || wx + N > M || wy + N > M) { free(W); return ORC_EINVAL; }
            for (int j = 0; j < n_sub; ++j)
                for (int i = 0; i < n_sub; ++i) {
                    double acc = 0.0;
                    for (int py = 0; py < N; ++py) {
                        double wyv = W[(size_t)j * N + py];
                        if (wyv == 0.0) continue;
                        for (int px = 0; px < N; ++px) {
                            double wxv = W[(size_t)i * N + px];
                            if (wxv == 0.0) continue;
                            acc += wyv * wxv * Iin[(size_t)(wy + py) * M + (wx + px)];
                        }
                    }
                    frame[(size_t)(qy * n_sub + j) * D + (qx * n_sub + i)] = acc;
                }
        }
    free(W);
    return ORC_OK;
}

/* O8: valid-subaperture mask from the pupil illumination,
 *   ill[j][i] = sum W[j][py] W[i][px] A^2[py][px];  valid iff
 *   ill >= thresh * b^2 * max(A^2)
 * (configs: "slopes over a >=50%-illumination mask"; reading A11: geometric,
 * `>=`, same mask for all four tiles).  Both sides are scaled by n_sub^2 so
 * that for binary A every quantity is an integer held exactly in a double.
 * Returns n_valid (>= 0) or a negative error. */
int orc_valid_mask(int N, int n_sub, const float *A, double thresh, unsigned char *valid) {
    if (n_sub < 1 || n_sub > N) return ORC_EINVAL;
    double *W = (double *)malloc(sizeof(double) * (size_t)n_sub * N);
    if (!W) return ORC_ENOMEM;
    orc_rebin_weights(N, n_sub, W);
    double amax2 = 0.0;
    for (size_t t = 0; t < (size_t)N * N; ++t) {
        double a2 = (double)A[t] * (double)A[t];
        if (a2 > amax2) amax2 = a2;
    }
    int count = 0;
    for (int j = 0; j < n_sub; ++j)
        for (int i = 0; i < n_sub; ++i) {
            double ill = 0.0;                  /* in units of 1/n_sub^2 px^2 */
            for (int py = 0; py < N; ++py) {
                double wy = W[(size_t)j * N + py] * (double)n_sub;
                if (wy == 0.0) continue;
                for (int px = 0; px < N; ++px) {
                    double wx = W[(size_t)i * N + px] * (double)n_sub;
                    if (wx == 0.0) continue;
                    double a = (double)A[(size_t)py * N + px];
                    ill += wy * wx * a * a;
                }
            }
            double full = (double)N * (double)N * amax2;   /* b^2 n_sub^2 max A^2 */
            int ok = (amax2 > 0.0) && (ill >= thresh * full);
            valid[(size_t)j * n_sub + i] = (unsigned char)ok;
            count += ok;
        }
    free(W);
    return count;
}

/* O9: quad-cell slopes over the valid subapertures.  With a, b, c, d the
 * tiles (qx,qy) = (0,0), (1,0), (0,1), (1,1) at subaperture (j,i):
 *   nbar = (1/n_valid) sum_valid (a+b+c+d)
 *   Sx = ((a+c) - (b+d)) / nbar,   Sy = ((a+b) - (c+d)) / nbar
 * output [Sx(valid, row-major) ..., Sy(valid, row-major) ...]; norm_mode 1
 * divides by the local a+b+c+d instead (reading A12: sign such that a +x
 * tilt gives Sx > 0).  (PAPER.md:L261-262 sc.in_pixels -> sc.out_slopes.) */
int orc_slopes(int n_sub, const double *frame, const unsigned char *valid, int norm_mode,
               double *slopes) {
    int D = 2 * n_sub;
    int nv = 0;
    double tot = 0.0;
    for (int j = 0; j < n_sub; ++j)
        for (int i = 0; i < n_sub; ++i)
            if (valid[(size_t)j * n_sub + i]) {
                double a = frame[(size_t)j * D + i], b = frame[(size_t)j * D + n_sub + i];
                double c = frame[(size_t)(n_sub + j) * D + i], d = frame[(size_t)(n_sub + j) * D + n_sub + i];
                tot += a + b + c + d;
                ++nv;
            }
    if (nv == 0) return ORC_EINVAL;
    double nbar = tot / (double)nv;
    int t = 0;
    for (int j = 0; j < n_sub; ++j)
        for (int i = 0; i < n_sub; ++i)
            if (valid[(size_t)j * n_sub + i]) {
                double a = frame[(size_t)j * D + i], b = frame[(size_t)j * D + n_sub + i];
                double c = frame[(size_t)(n_sub + j) * D + i], d = frame[(size_t)(n_sub + j) * D + n_sub + i];
                double den = (norm_mode == 1) ? (a + b + c + d) : nbar;
                slopes[t] = ((a + c) - (b + d)) / den;
                slopes[nv + t] = ((a + b) - (c + d)) / den;
                ++t;
            }
    return nv;
}

/* Whole path O0..O9 for a batch of B phase screens (float32 [B][N][N]).
 * frames: double [B][2n_sub][2n_sub]; slopes: double [B][2 n_valid] (may be
 * NULL).  s <= 0 selects the default M/4.  Returns n_valid or an error. */
int orc_pwfs_run(int N, int M, const float *A, int s, double r, int K, double theta0,
                 int n_sub, double thresh, int norm_mode, int B, const float *phase,
                 double *frames, double *slopes) {
    if (N < 2 || M < 2 * N || (M & 1) || K < 1 || r < 0.0 || B < 0) return ORC_EINVAL;
    if (s <= 0) { if (M % 4) return ORC_EINVAL; s = M / 4; }
    if (2 * s < N || s > M / 2 - N / 2) return ORC_EINVAL;
    size_t MM = (size_t)M * M;
    int D = 2 * n_sub;
    unsigned char *valid = (unsigned char *)malloc((size_t)n_sub * n_sub);
    zc *mask = (zc *)malloc(sizeof(zc) * MM);
    double *Ifull = (double *)malloc(sizeof(double) * MM);
    if (!valid || !mask || !Ifull) { free(valid); free(mask); free(Ifull); return ORC_ENOMEM; }
    int nv = orc_valid_mask(N, n_sub, A, thresh, valid);            /* O8 */
    int rc = (nv > 0) ? ORC_OK : ORC_EINVAL;
    if (!rc) orc_pyramid_mask(M, (double)s, mask);                  /* O4 */
    for (int bb = 0; bb < B && !rc; ++bb) {
        rc = orc_intensity(N, M, A, phase + (size_t)bb * N * N, K, r, theta0, mask, Ifull, 0);
        if (!rc) rc = orc_frame(N, M, s, n_sub, Ifull, frames + (size_t)bb * D * D);   /* O7 */
        if (!rc && slopes) {
            int n2 = orc_slopes(n_sub, frames + (size_t)bb * D * D, valid, norm_mode,
                                slopes + (size_t)bb * 2 * nv);      /* O9 */
            if (n2 != nv) rc = ORC_EINVAL;
        }
    }
    free(valid); free(mask); free(Ifull);
    return rc ? rc : nv;
}

/* Whole path with the f3 generalisations: tilt list (dx,dy,w) in lambda/D in
 * place of the circle and an optional square field stop of half-width
 * stop_h focal-plane bins (< 0: none).  Otherwise identical to orc_pwfs_run. */
int orc_pwfs_run_list(int N, int M, const float *A, int s, int n_pts, const double *dx,
                      const double *dy, const double *w, double stop_h, int n_sub, double thresh,
                      int norm_mode, int B, const float *phase, double *frames, double *slopes) {
    if (N < 2 || M < 2 * N || (M & 1) || n_pts < 1 || B < 0) return ORC_EINVAL;
    if (s <= 0) { if (M % 4) return ORC_EINVAL; s = M / 4; }
    if (2 * s < N || s > M / 2 - N / 2) return ORC_EINVAL;
    size_t MM = (size_t)M * M;
    int D = 2 * n_sub;
    unsigned char *valid = (unsigned char *)malloc((size_t)n_sub * n_sub);
    zc *mask = (zc *)malloc(sizeof(zc) * MM);
    double *Ifull = (double *)malloc(sizeof(double) * MM);
    if (!valid || !mask || !Ifull) { free(valid); free(mask); free(Ifull); return ORC_ENOMEM; }
    int nv = orc_valid_mask(N, n_sub, A, thresh, valid);            /* O8 */
    int rc = (nv > 0) ? ORC_OK : ORC_EINVAL;
    if (!rc) {
        orc_pyramid_mask(M, (double)s, mask);                       /* O4 */
        orc_field_stop(M, stop_h, mask);                            /* f3 */
    }
    for (int bb = 0; bb < B && !rc; ++bb) {
        rc = orc_intensity_list(N, M, A, phase + (size_t)bb * N * N, n_pts, dx, dy, w, mask, Ifull, 0);
        if (!rc) rc = orc_frame(N, M, s, n_sub, Ifull, frames + (size_t)bb * D * D);   /* O7 */
        if (!rc && slopes) {
            int n2 = orc_slopes(n_sub, frames + (size_t)bb * D * D, valid, norm_mode,
                                slopes + (size_t)bb * 2 * nv);      /* O9 */
            if (n2 != nv) rc = ORC_EINVAL;
        }
    }
    free(valid); free(mask); free(Ifull);
    return rc ? rc : nv;
}
