/*
 * pyr_oracle.c -- CPU oracle for the modulated pyramid wavefront-sensor propagation.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no source, header, table or helper with the CUDA library (libpyr).
 *
 * What it is: the plain definition of the path named by BASELINE.json:north_star
 * (in the paper: the `ModulatedPyramid` processing object followed by `PyrSlopec`,
 * PAPER.md:316-317, 327 (Table 4), parameterised as in Listing 2, PAPER.md:528-556,
 * 592-604, with the FFT workload n_mod x N_fft x N_fft of Table 2),
 * written out step by step in double precision with its own DFT/FFT, in the order and
 * notation of SURVEY.md section 8(c):
 *
 *   1. theta_k = 2 pi k / M,  (a_kx, a_ky) = r (cos theta_k, sin theta_k)
 *   2. E_k[y+o][x+o] = A[y][x] exp(i (phi[y][x] + (2 pi / P)(a_kx (x-c_p) + a_ky (y-c_p)))),
 *      o = (N-P)/2, c_p = (P-1)/2, zero elsewhere in the N x N array
 *   3. F_k = DFT2(E_k), sign -, unnormalised
 *   4. G_k = F_k * mask,  mask[v][u] = (-i)^(|f(u)|+|f(v)|), f(u) = u (u < N/2) else u-N
 *   5. O_k = IDFT2(G_k), sign +, scaled 1/N^2
 *   6. I = sum_k |O_k|^2
 *   7. D[Y][X] = sum over b x b blocks of I
 *   8-10. quadrants Qa,Qb,Qc,Qd of D, validity map, global-mean normalised slopes.
 *
 * The paper itself prints no formula for the sensor (reading S1); the
 * readings S2-S16 listed there and in DESIGN.md are the ones implemented here.
 * No blocking, pruning, separability or symmetry shortcut is used: every modulation point
 * does two full N x N 2-D transforms of the whole padded array (radix-2 FFT lines when N is a
 * power of two, textbook mixed-radix Cooley-Tukey lines otherwise -- the paper's own sizes 660 and
 * 1600 -- pinned against the direct O(N^2) DFT pyro_dft_direct, which stays exported for that).
 *
 * Parity pins (tests/test_oracle_pins.py, all `-m "not gpu"`): brute-force O(N^4) DFT chain
 * written independently in NumPy, closed-form 1-D DFTs, numpy.fft as a library cross-check
 * of the FFT routine, Parseval, identity mask, pure-shift mask, flat-wavefront symmetry,
 * tilt sign/linearity, translation and dihedral equivariance, integer focal shift, and the
 * separable-operator identity.  No function here is "parity unpinned" with respect to the
 * definition above; agreement with the SPECULA/PASSATA *implementations* is unpinned
 * (their code and data are not available; SURVEY.md 8(c) last row).
 *
 * Build: gcc -O2 -fPIC -shared -pthread -o liboracle.so pyr_oracle.c -lm
 */
#include <math.h>
#include <pthread.h>
#include <stdlib.h>
#include <string.h>

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

/* ------------------------------------------------------------------ 1-D transforms */

/* Direct O(n^2) DFT, any n >= 1.  out[u] = sum_x in[x] exp(sign * 2 pi i u x / n).
 * Arrays are interleaved (re, im).  No scaling.  The phase index (u*x mod n) is reduced
 * in integers so the argument of sin/cos stays in [0, 2 pi). */
void pyro_dft_direct(int n, int sign, const double *in, double *out)
{
    for (int u = 0; u < n; ++u) {
        double sr = 0.0, si = 0.0;
        for (int x = 0; x < n; ++x) {
            long long m = ((long long)u * x) % n;
            double ang = (double)sign * 2.0 * M_PI * (double)m / (double)n;
            double c = cos(ang), s = sin(ang);
            sr += in[2 * x] * c - in[2 * x + 1] * s;
            si += in[2 * x] * s + in[2 * x + 1] * c;
        }
        out[2 * u] = sr;
        out[2 * u + 1] = si;
    }
}

/* Twiddle table w[j] = exp(sign * 2 pi i j / n), j < n/2, each from a direct sin/cos call
 * (no recurrence). */
static void make_twiddles(int n, int sign, double *w)
{
    for (int j = 0; j < n / 2; ++j) {
        double ang = (double)sign * 2.0 * M_PI * (double)j / (double)n;
        w[2 * j] = cos(ang);
        w[2 * j + 1] = sin(ang);
    }
}

/* In-place iterative radix-2 decimation-in-time FFT, n a power of two, unscaled.
 * `w` is make_twiddles(n, sign).  Textbook Cooley-Tukey: bit-reversal permutation, then
 * log2(n) butterfly stages. */
static void fft_pow2(int n, double *a, const double *w)
{
    for (int i = 1, j = 0; i < n; ++i) {
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) {
            double tr = a[2 * i], ti = a[2 * i + 1];
            a[2 * i] = a[2 * j];
            a[2 * i + 1] = a[2 * j + 1];
            a[2 * j] = tr;
            a[2 * j + 1] = ti;
        }
    }
    for (int len = 2; len <= n; len <<= 1) {
        int half = len >> 1, step = n / len;
        for (int i = 0; i < n; i += len) {
            for (int j = 0; j < half; ++j) {
                double wr = w[2 * (j * step)], wi = w[2 * (j * step) + 1];
                double *p = a + 2 * (i + j), *q = a + 2 * (i + j + half);
                double xr = q[0] * wr - q[1] * wi;
                double xi = q[0] * wi + q[1] * wr;
                q[0] = p[0] - xr;
                q[1] = p[1] - xi;
                p[0] += xr;
                p[1] += xi;
            }
        }
    }
}

static int is_pow2(int n) { return n >= 1 && (n & (n - 1)) == 0; }

/* 2-D transform of a row-major n x n complex array, in place, unscaled: every row, then
 * every column (a column is gathered into `col`, transformed, scattered back). */
static void fft2d_pow2(int n, double *a, const double *w, double *col)
{
    for (int y = 0; y < n; ++y) fft_pow2(n, a + 2 * (size_t)y * n, w);
    for (int x = 0; x < n; ++x) {
        for (int y = 0; y < n; ++y) {
            col[2 * y] = a[2 * ((size_t)y * n + x)];
            col[2 * y + 1] = a[2 * ((size_t)y * n + x) + 1];
        }
        fft_pow2(n, col, w);
        for (int y = 0; y < n; ++y) {
            a[2 * ((size_t)y * n + x)] = col[2 * y];
            a[2 * ((size_t)y * n + x) + 1] = col[2 * y + 1];
        }
    }
}

/* Any n (the paper's own FFT sizes, 660 = 2^2 3 5 11 and 1600 = 2^6 5^2, are not powers of two;
 * PAPER.md:193, 195): the textbook mixed-radix Cooley-Tukey recursion, decimation in time.  With p the
 * smallest prime factor of n and m = n / p,
 *     X[k + q m] = sum_{r<p} W_p^(r q) ( W_n^(r k) Y_r[k] ),   Y_r = DFT_m( x[r], x[r + p], ... ),
 * and a prime length is the direct O(n^2) sum.  W_n^j = exp(sign 2 pi i j / n) comes from a table of
 * the top-level length n0 (each entry from a direct sin/cos call; every index reduced mod n0 in
 * integers).  Exact DFT up to rounding; pinned against pyro_dft_direct and the closed forms (P2). */
static void make_table_full(int n, int sign, double *w /* [n][2] */)
{
    for (int j = 0; j < n; ++j) {
        double ang = (double)sign * 2.0 * M_PI * (double)j / (double)n;
        w[2 * j] = cos(ang);
        w[2 * j + 1] = sin(ang);
    }
}

static int smallest_prime_factor(int n)
{
    for (int p = 2; (long long)p * p <= n; ++p)
        if (n % p == 0) return p;
    return n;
}

/* out[0..n) = DFT_n of in[0], in[is], in[2 is], ...; w = table of length n0, n | n0; tmp: n0 complex. */
static void fft_mixed_rec(int n, const double *in, int is, double *out, const double *w, int n0, double *tmp)
{
    if (n == 1) { out[0] = in[0]; out[1] = in[1]; return; }
    const int ws = n0 / n;                      /* W_n^j = w[(j mod n) * ws] */
    const int p = smallest_prime_factor(n), m = n / p;
    if (p == n) {                               /* prime length: the direct sum */
        for (int u = 0; u < n; ++u) {
            double sr = 0.0, si = 0.0;
            long long e = 0;                    /* (u x) mod n */
            for (int x = 0; x < n; ++x) {
                const double c = w[2 * e * ws], sn = w[2 * e * ws + 1];
                const double xr = in[2 * (size_t)x * is], xi = in[2 * (size_t)x * is + 1];
                sr += xr * c - xi * sn;
                si += xr * sn + xi * c;
                e += u; if (e >= n) e -= n;
            }
            out[2 * u] = sr; out[2 * u + 1] = si;
        }
        return;
    }
    for (int r = 0; r < p; ++r)                 /* Y_r -> out[r m .. r m + m) */
        fft_mixed_rec(m, in + 2 * (size_t)r * is, is * p, out + 2 * (size_t)r * m, w, n0, tmp);
    for (int k = 0; k < m; ++k) {
        for (int r = 0; r < p; ++r) {           /* t_r = W_n^(r k) Y_r[k] */
            const long long e = ((long long)r * k) % n;
            const double c = w[2 * e * ws], sn = w[2 * e * ws + 1];
            const double yr = out[2 * ((size_t)r * m + k)], yi = out[2 * ((size_t)r * m + k) + 1];
            tmp[2 * r] = yr * c - yi * sn;
            tmp[2 * r + 1] = yr * sn + yi * c;
        }
        for (int q = 0; q < p; ++q) {           /* X[k + q m] = sum_r W_p^(r q) t_r */
            double sr = 0.0, si = 0.0;
            for (int r = 0; r < p; ++r) {
                const long long e = ((long long)r * q) % p;
                const double c = w[2 * e * (n0 / p)], sn = w[2 * e * (n0 / p) + 1];
                sr += tmp[2 * r] * c - tmp[2 * r + 1] * sn;
                si += tmp[2 * r] * sn + tmp[2 * r + 1] * c;
            }
            out[2 * ((size_t)k + (size_t)q * m)] = sr;
            out[2 * ((size_t)k + (size_t)q * m) + 1] = si;
        }
    }
}

/* One line of n complex numbers: out = DFT_n(in), out must not alias in; tmp: n complex. */
static void fft_mixed_line(int n, const double *wfull, const double *in, double *out, double *tmp)
{
    fft_mixed_rec(n, in, 1, out, wfull, n, tmp);
}

/* 2-D transform for any n: every row, then every column, each by the mixed-radix line transform.
 * `col`, `tmp` and `tmp2` are scratch lines of n complex numbers. */
static void fft2d_mixed(int n, double *a, const double *wfull, double *col, double *tmp, double *tmp2)
{
    for (int y = 0; y < n; ++y) {
        fft_mixed_line(n, wfull, a + 2 * (size_t)y * n, tmp, tmp2);
        memcpy(a + 2 * (size_t)y * n, tmp, sizeof(double) * 2 * (size_t)n);
    }
    for (int x = 0; x < n; ++x) {
        for (int y = 0; y < n; ++y) {
            col[2 * y] = a[2 * ((size_t)y * n + x)];
            col[2 * y + 1] = a[2 * ((size_t)y * n + x) + 1];
        }
        fft_mixed_line(n, wfull, col, tmp, tmp2);
        for (int y = 0; y < n; ++y) {
            a[2 * ((size_t)y * n + x)] = tmp[2 * y];
            a[2 * ((size_t)y * n + x) + 1] = tmp[2 * y + 1];
        }
    }
}

/* Exported 1-D transform: radix-2 FFT for powers of two, mixed-radix FFT otherwise.  In place, unscaled.
 * Returns 0, or 1 on bad arguments / allocation failure. */
int pyro_fft1d(int n, int sign, double *a)
{
    if (n < 1 || (sign != 1 && sign != -1) || !a) return 1;
    if (n == 1) return 0;
    if (is_pow2(n)) {
        double *w = (double *)malloc(sizeof(double) * (size_t)n);
        if (!w) return 1;
        make_twiddles(n, sign, w);
        fft_pow2(n, a, w);
        free(w);
    } else {
        double *t = (double *)malloc(sizeof(double) * 2 * (size_t)n);
        double *w = (double *)malloc(sizeof(double) * 2 * (size_t)n);
        double *tmp = (double *)malloc(sizeof(double) * 2 * (size_t)n);
        if (!t || !w || !tmp) { free(t); free(w); free(tmp); return 1; }
        make_table_full(n, sign, w);
        fft_mixed_line(n, w, a, t, tmp);
        memcpy(a, t, sizeof(double) * 2 * (size_t)n);
        free(t); free(w); free(tmp);
    }
    return 0;
}

/* Exported 2-D transform of an n x n array: radix-2 FFT for powers of two, mixed radix otherwise. */
int pyro_fft2d(int n, int sign, double *a)
{
    if (n < 1 || (sign != 1 && sign != -1) || !a) return 1;
    double *w = (double *)malloc(sizeof(double) * 2 * (size_t)(n > 1 ? n : 2));
    double *col = (double *)malloc(sizeof(double) * 2 * (size_t)n);
    double *tmp = (double *)malloc(sizeof(double) * 2 * (size_t)n);
    double *tmp2 = (double *)malloc(sizeof(double) * 2 * (size_t)n);
    if (!w || !col || !tmp || !tmp2) { free(w); free(col); free(tmp); free(tmp2); return 1; }
    if (is_pow2(n)) {
        make_twiddles(n, sign, w);
        fft2d_pow2(n, a, w, col);
    } else {
        make_table_full(n, sign, w);
        fft2d_mixed(n, a, w, col, tmp, tmp2);
    }
    free(w);
    free(col);
    free(tmp);
    free(tmp2);
    return 0;
}

/* ------------------------------------------------------------------ the sensor */

/* Step 4: mask[v][u] = (-i)^e, e = (|f(u)| + |f(v)|) mod 4, evaluated exactly from the
 * integer exponent.  (-i)^0 = 1, (-i)^1 = -i, (-i)^2 = -1, (-i)^3 = i. */
static int absfreq(int u, int n) { return u < n / 2 ? u : n - u; }

void pyro_pyramid_mask(int n, double *mask /* [n][n][2] */)
{
    static const double re[4] = {1.0, 0.0, -1.0, 0.0};
    static const double im[4] = {0.0, -1.0, 0.0, 1.0};
    for (int v = 0; v < n; ++v)
        for (int u = 0; u < n; ++u) {
            int e = (absfreq(u, n) + absfreq(v, n)) & 3;
            mask[2 * ((size_t)v * n + u)] = re[e];
            mask[2 * ((size_t)v * n + u) + 1] = im[e];
        }
}

typedef struct {
    int P, N, M, B;
    double r;
    const float *amp, *phase;
    const double *mask;   /* [N][N][2] */
    const double *ax, *ay, *w;  /* NULL: the modulation circle of step 1; else M points (lambda/D) and weights (w NULL = 1) */
    const double *ps;           /* NULL, or per-point factor on the whole pupil phase (polychromatic sensor: lambda_0 / lambda) */
    int double_roof;            /* two roof prisms in two focal planes instead of the four-face mask */
    double kappa;               /* ... with the pupil-plane factor exp(i pi kappa rho^2) of the propagation between them */
    int tid, nthreads;
    double *I;            /* this worker's accumulator, [B][N][N], zero-initialised */
    int err;
} worker_t;

/* One worker handles the (source, k) tasks with task index == tid (mod nthreads), in
 * increasing order.  Steps 1-6 for each task. */
static void *worker_main(void *arg)
{
    worker_t *wk = (worker_t *)arg;
    const int P = wk->P, N = wk->N, M = wk->M, B = wk->B;
    const size_t NN = (size_t)N * N;
    const int o = (N - P) / 2;
    const double cp = 0.5 * (double)(P - 1);
    double *E = (double *)malloc(sizeof(double) * 2 * NN);
    const int p2 = is_pow2(N);
    double *wf = (double *)malloc(sizeof(double) * 2 * (size_t)(N > 1 ? N : 2));
    double *wi = (double *)malloc(sizeof(double) * 2 * (size_t)(N > 1 ? N : 2));
    double *col = (double *)malloc(sizeof(double) * 2 * (size_t)N);
    double *tmp = (double *)malloc(sizeof(double) * 2 * (size_t)N);
    double *tmp2 = (double *)malloc(sizeof(double) * 2 * (size_t)N);
    if (!E || !wf || !wi || !col || !tmp || !tmp2) {
        wk->err = 1; free(E); free(wf); free(wi); free(col); free(tmp); free(tmp2); return NULL;
    }
    if (p2) {
        make_twiddles(N, -1, wf);
        make_twiddles(N, +1, wi);
    } else {
        make_table_full(N, -1, wf);
        make_table_full(N, +1, wi);
    }
    const double inv = 1.0 / ((double)N * (double)N);

    for (int task = wk->tid; task < B * M; task += wk->nthreads) {
        const int s = task / M, k = task % M;
        /* step 1 (or, for pyr_oracle_compute_points, the given point and weight) */
        double akx, aky, wgt = 1.0, psc = 1.0;
        if (wk->ax) {
            akx = wk->ax[k]; aky = wk->ay[k];
            if (wk->w) wgt = wk->w[k];
            if (wk->ps) psc = wk->ps[k];
        } else {
            const double theta = 2.0 * M_PI * (double)k / (double)M;
            akx = wk->r * cos(theta); aky = wk->r * sin(theta);
        }
        /* step 2 */
        memset(E, 0, sizeof(double) * 2 * NN);
        for (int y = 0; y < P; ++y)
            for (int x = 0; x < P; ++x) {
                double A = (double)wk->amp[((size_t)s * P + y) * P + x];
                double ph = (double)wk->phase[((size_t)s * P + y) * P + x];
                double tilt = (2.0 * M_PI / (double)P) * (akx * ((double)x - cp) + aky * ((double)y - cp));
                double *e = E + 2 * ((size_t)(y + o) * N + (x + o));
                e[0] = A * cos(psc * (ph + tilt));
                e[1] = A * sin(psc * (ph + tilt));
            }
        /* step 3 */
        if (p2) fft2d_pow2(N, E, wf, col); else fft2d_mixed(N, E, wf, col, tmp, tmp2);
        if (wk->double_roof) {
            /* ModulatedDoubleRoof (reading DR1 of DESIGN.md section 15): roof 1 splits along x in
             * the first focal plane, mask1[v][u] = (-i)^|f(u)|; back to the pupil plane (inverse 2-D DFT, 1/N^2);
             * the propagation to the second focal plane is the factor q[y][x] = exp(i pi kappa ((x-c)^2 + (y-c)^2)),
             * c = (N-1)/2; forward 2-D DFT; roof 2 splits along y, mask2[v][u] = (-i)^|f(v)|. */
            static const double re[4] = {1.0, 0.0, -1.0, 0.0}, im[4] = {0.0, -1.0, 0.0, 1.0};
            const double c = 0.5 * (double)(N - 1);
            for (int v = 0; v < N; ++v)
                for (int u = 0; u < N; ++u) {
                    const int ex = absfreq(u, N) & 3;
                    double *f = E + 2 * ((size_t)v * N + u);
                    const double fr = f[0], fi = f[1];
                    f[0] = fr * re[ex] - fi * im[ex];
                    f[1] = fr * im[ex] + fi * re[ex];
                }
            if (p2) fft2d_pow2(N, E, wi, col); else fft2d_mixed(N, E, wi, col, tmp, tmp2);
            for (int y = 0; y < N; ++y)
                for (int x = 0; x < N; ++x) {
                    const double rho2 = ((double)x - c) * ((double)x - c) + ((double)y - c) * ((double)y - c);
                    const double qr = cos(M_PI * wk->kappa * rho2), qi = sin(M_PI * wk->kappa * rho2);
                    double *f = E + 2 * ((size_t)y * N + x);
                    const double fr = f[0] * inv, fi = f[1] * inv;
                    f[0] = fr * qr - fi * qi;
                    f[1] = fr * qi + fi * qr;
                }
            if (p2) fft2d_pow2(N, E, wf, col); else fft2d_mixed(N, E, wf, col, tmp, tmp2);
            for (int v = 0; v < N; ++v)
                for (int u = 0; u < N; ++u) {
                    const int ey = absfreq(v, N) & 3;
                    double *f = E + 2 * ((size_t)v * N + u);
                    const double fr = f[0], fi = f[1];
                    f[0] = fr * re[ey] - fi * im[ey];
                    f[1] = fr * im[ey] + fi * re[ey];
                }
        } else
        /* step 4 */
        for (size_t i = 0; i < NN; ++i) {
            double fr = E[2 * i], fi = E[2 * i + 1];
            double mr = wk->mask[2 * i], mi = wk->mask[2 * i + 1];
            E[2 * i] = fr * mr - fi * mi;
            E[2 * i + 1] = fr * mi + fi * mr;
        }
        /* step 5 */
        if (p2) fft2d_pow2(N, E, wi, col); else fft2d_mixed(N, E, wi, col, tmp, tmp2);
        /* step 6 */
        double *I = wk->I + (size_t)s * NN;
        for (size_t i = 0; i < NN; ++i) {
            double orr = E[2 * i] * inv, oi = E[2 * i + 1] * inv;
            I[i] += wgt * (orr * orr + oi * oi);
        }
    }
    free(E); free(wf); free(wi); free(col); free(tmp); free(tmp2);
    return NULL;
}

/* Default validity map (step 9): (Y,X) valid iff (2Y-(Nq-1))^2 + (2X-(Nq-1))^2 <= ns^2,
 * ns = P/b; integer test. */
void pyro_default_valid(int P, int N, int b, unsigned char *valid /* [Nq][Nq] */)
{
    const int Nq = N / b / 2, ns = P / b;
    for (int Y = 0; Y < Nq; ++Y)
        for (int X = 0; X < Nq; ++X) {
            long long dy = 2 * Y - (Nq - 1), dx = 2 * X - (Nq - 1);
            valid[(size_t)Y * Nq + X] = (dy * dy + dx * dx <= (long long)ns * ns) ? 1 : 0;
        }
}

/* Steps 7: D[Y][X] = sum_{j<b} sum_{i<b} I[bY+j][bX+i]. */
void pyro_rebin(int N, int b, const double *I /* [N][N] */, double *D /* [N/b][N/b] */)
{
    const int Nd = N / b;
    for (int Y = 0; Y < Nd; ++Y)
        for (int X = 0; X < Nd; ++X) {
            double s = 0.0;
            for (int j = 0; j < b; ++j)
                for (int i = 0; i < b; ++i) s += I[(size_t)(b * Y + j) * N + (b * X + i)];
            D[(size_t)Y * Nd + X] = s;
        }
}

/* Steps 8-10 for one source.  slopes = [2][Nq][Nq], plane 0 = sx, plane 1 = sy.
 * If no pixel is valid, or the mean total is 0, all slopes are 0. */
void pyro_slopes(int Nd, const double *D, const unsigned char *valid, double *slopes)
{
    const int Nq = Nd / 2;
    double tot = 0.0;
    long long nv = 0;
    for (int Y = 0; Y < Nq; ++Y)
        for (int X = 0; X < Nq; ++X)
            if (valid[(size_t)Y * Nq + X]) {
                double Qa = D[(size_t)Y * Nd + X], Qb = D[(size_t)Y * Nd + X + Nq];
                double Qc = D[(size_t)(Y + Nq) * Nd + X], Qd = D[(size_t)(Y + Nq) * Nd + X + Nq];
                tot += Qa + Qb + Qc + Qd;
                ++nv;
            }
    double Tbar = nv > 0 ? tot / (double)nv : 0.0;
    for (int Y = 0; Y < Nq; ++Y)
        for (int X = 0; X < Nq; ++X) {
            double sx = 0.0, sy = 0.0;
            if (valid[(size_t)Y * Nq + X] && Tbar > 0.0) {
                double Qa = D[(size_t)Y * Nd + X], Qb = D[(size_t)Y * Nd + X + Nq];
                double Qc = D[(size_t)(Y + Nq) * Nd + X], Qd = D[(size_t)(Y + Nq) * Nd + X + Nq];
                sx = ((Qb + Qd) - (Qa + Qc)) / Tbar;
                sy = ((Qc + Qd) - (Qa + Qb)) / Tbar;
            }
            slopes[(size_t)Y * Nq + X] = sx;
            slopes[(size_t)Nq * Nq + (size_t)Y * Nq + X] = sy;
        }
}

/*
 * The whole path.  All pointers are host memory.
 *   amp, phase : float32 [B][P][P] (converted to double here, so input rounding is shared
 *                with the GPU side)
 *   mask       : NULL for the four-face pyramid of step 4, else [N][N][2] doubles
 *   valid      : NULL for the default map, else [Nq][Nq] bytes
 *   I_full     : NULL or [B][N][N] doubles (full-resolution intensity, step 6)
 *   D          : NULL or [B][Nd][Nd]
 *   slopes     : NULL or [B][2][Nq][Nq]
 *   nthreads   : >= 1 worker threads over the (source, k) tasks; the result does not depend
 *                on it beyond the summation order of the per-worker accumulators.
 * Returns 0 on success, 1 bad arguments, 3 out of memory.
 */
static int compute_impl(int P, int N, int M, double r, const double *ax, const double *ay, const double *w,
                        const double *ps, int double_roof, double kappa,
                        int b, int B, const float *amp, const float *phase,
                        const double *mask, const unsigned char *valid,
                        double *I_full, double *D, double *slopes, int nthreads)
{
    if (N < 2 || (N & 1) || P < 1 || P > N || ((N - P) & 1) || M < 1 || b < 1 || B < 1 ||
        (N % b) != 0 || ((N / b) & 1) || !amp || !phase || nthreads < 1 || !(r >= 0.0))
        return 1;
    const size_t NN = (size_t)N * N;
    const int Nd = N / b, Nq = Nd / 2;
    if (nthreads > B * M) nthreads = B * M;

    double *mk = NULL;
    if (!mask) {
        mk = (double *)malloc(sizeof(double) * 2 * NN);
        if (!mk) return 3;
        pyro_pyramid_mask(N, mk);
        mask = mk;
    }
    worker_t *wk = (worker_t *)calloc((size_t)nthreads, sizeof(worker_t));
    pthread_t *th = (pthread_t *)calloc((size_t)nthreads, sizeof(pthread_t));
    int rc = 0;
    if (!wk || !th) { rc = 3; goto done; }
    for (int t = 0; t < nthreads; ++t) {
        wk[t].P = P; wk[t].N = N; wk[t].M = M; wk[t].B = B; wk[t].r = r;
        wk[t].amp = amp; wk[t].phase = phase; wk[t].mask = mask;
        wk[t].ax = ax; wk[t].ay = ay; wk[t].w = w;
        wk[t].ps = ps; wk[t].double_roof = double_roof; wk[t].kappa = kappa;
        wk[t].tid = t; wk[t].nthreads = nthreads;
        wk[t].I = (double *)calloc((size_t)B * NN, sizeof(double));
        if (!wk[t].I) rc = 3;
    }
    if (rc == 0) {
        for (int t = 1; t < nthreads; ++t) pthread_create(&th[t], NULL, worker_main, &wk[t]);
        worker_main(&wk[0]);
        for (int t = 1; t < nthreads; ++t) pthread_join(th[t], NULL);
        for (int t = 0; t < nthreads; ++t) if (wk[t].err) rc = 3;
    }
    if (rc == 0) {
        /* sum the per-worker accumulators in worker order into worker 0's */
        double *I = wk[0].I;
        for (int t = 1; t < nthreads; ++t)
            for (size_t i = 0; i < (size_t)B * NN; ++i) I[i] += wk[t].I[i];
        if (I_full) memcpy(I_full, I, sizeof(double) * (size_t)B * NN);
        if (D || slopes) {
            double *Dd = (double *)malloc(sizeof(double) * (size_t)Nd * Nd);
            unsigned char *vm = (unsigned char *)malloc((size_t)(Nq > 0 ? Nq * Nq : 1));
            if (!Dd || !vm) rc = 3;
            else {
                if (valid) memcpy(vm, valid, (size_t)Nq * Nq);
                else pyro_default_valid(P, N, b, vm);
                for (int s = 0; s < B; ++s) {
                    pyro_rebin(N, b, I + (size_t)s * NN, Dd);
                    if (D) memcpy(D + (size_t)s * Nd * Nd, Dd, sizeof(double) * (size_t)Nd * Nd);
                    if (slopes) pyro_slopes(Nd, Dd, vm, slopes + (size_t)s * 2 * Nq * Nq);
                }
            }
            free(Dd); free(vm);
        }
    }
done:
    if (wk) for (int t = 0; t < nthreads; ++t) free(wk[t].I);
    free(wk); free(th); free(mk);
    return rc;
}

int pyr_oracle_compute(int P, int N, int M, double r, int b, int B,
                       const float *amp, const float *phase,
                       const double *mask, const unsigned char *valid,
                       double *I_full, double *D, double *slopes, int nthreads)
{
    return compute_impl(P, N, M, r, NULL, NULL, NULL, NULL, 0, 0.0, b, B, amp, phase, mask, valid, I_full, D, slopes, nthreads);
}

/* The same path for an arbitrary list of modulation points instead of the circle of step 1
 * (pyr_plan_create_points; extended sources and other modulation paths):
 * I = sum_k w[k] |O_k|^2 with the tilt (ax[k], ay[k]) in lambda/D; w == NULL means weight 1.
 * Returns 1 as well if a weight is negative. */
int pyr_oracle_compute_points(int P, int N, int M, const double *ax, const double *ay, const double *w,
                              int b, int B, const float *amp, const float *phase,
                              const double *mask, const unsigned char *valid,
                              double *I_full, double *D, double *slopes, int nthreads)
{
    if (!ax || !ay || M < 1) return 1;
    if (w) for (int k = 0; k < M; ++k) if (!(w[k] >= 0.0)) return 1;
    return compute_impl(P, N, M, 0.0, ax, ay, w, NULL, 0, 0.0, b, B, amp, phase, mask, valid, I_full, D, slopes, nthreads);
}

/* PolyCromPyramid (reading PC1 of DESIGN.md section 15): the sensor sums the intensities of
 * n_wl wavelengths.  amp and phase are given at the reference wavelength lambda_0; at wavelength l the optical
 * path is the same, so the whole pupil phase -- turbulence and modulation tilt alike -- is scaled by
 * ratio[l] = lambda_0 / lambda_l, the sampling (P, N) and the mask (a fixed pupil-image separation) stay:
 *   E_{k,l} = A exp(i ratio[l] (phi + tilt_k)),   I = sum_l weight[l] sum_k |O_{k,l}|^2,
 * with the modulation circle (M, r in lambda_0 / D) of step 1.  weight NULL = 1. */
int pyr_oracle_compute_poly(int P, int N, int M, double r, int n_wl, const double *ratio, const double *weight,
                            int b, int B, const float *amp, const float *phase,
                            const double *mask, const unsigned char *valid,
                            double *I_full, double *D, double *slopes, int nthreads)
{
    if (n_wl < 1 || !ratio || M < 1 || !(r >= 0.0)) return 1;
    if (weight) for (int l = 0; l < n_wl; ++l) if (!(weight[l] >= 0.0)) return 1;
    const int MM = M * n_wl;
    double *ax = (double *)malloc(sizeof(double) * 4 * (size_t)MM);
    if (!ax) return 3;
    double *ay = ax + MM, *w = ay + MM, *ps = w + MM;
    for (int l = 0; l < n_wl; ++l)
        for (int k = 0; k < M; ++k) {
            const double theta = 2.0 * M_PI * (double)k / (double)M;
            ax[l * M + k] = r * cos(theta);
            ay[l * M + k] = r * sin(theta);
            w[l * M + k] = weight ? weight[l] : 1.0;
            ps[l * M + k] = ratio[l];
        }
    const int rc = compute_impl(P, N, MM, 0.0, ax, ay, w, ps, 0, 0.0, b, B, amp, phase, mask, valid, I_full, D, slopes, nthreads);
    free(ax);
    return rc;
}

/* ModulatedDoubleRoof: the path of pyr_oracle_compute with the two-plane roof masks described in worker_main
 * in place of step 4.  kappa = 0 puts both roof edges in the same focal plane. */
int pyr_oracle_compute_double_roof(int P, int N, int M, double r, double kappa, int b, int B,
                                   const float *amp, const float *phase, const unsigned char *valid,
                                   double *I_full, double *D, double *slopes, int nthreads)
{
    return compute_impl(P, N, M, r, NULL, NULL, NULL, NULL, 1, kappa, b, B, amp, phase, NULL, valid, I_full, D, slopes, nthreads);
}
