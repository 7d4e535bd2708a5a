/*
 * sh_oracle.c -- CPU oracle for the Shack-Hartmann spot-and-centroid path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/ and bench.py's extras may build,
 * load or call it.  It shares no source, header, table or helper with the CUDA library.
 *
 * What it is: the second FFT workload of the paper: the `SH` processing
 * object followed by `ShSlopec` (Table 4), whose cost the paper states as
 * "n_subapertures x FFT x FFT" (Table 2: 314x56x56, 1256x68x68, 6x3630x240x240, PAPER.md:194,
 * 196-197).  The paper prints no formula for it either; the textbook Fourier-optics lenslet model
 * is written out below in double precision, with the readings listed in DESIGN.md section 12:
 *
 *   1. n_sub x n_sub lenslets over the P x P pupil, p = P / n_sub pixels each; sub-aperture
 *      (sy, sx) sees e[y][x] = A exp(i phi) at pupil pixel (sy p + y, sx p + x), 0 <= y, x < p.
 *   2. f[v][u] = sum_{y,x<p} e[y][x] exp(-2 pi i (u x + v y) / F): the F x F DFT of the patch
 *      zero-padded to F x F (sign -, unnormalised).
 *   3. S[v][u] = |f[v][u]|^2 / F^2 (so that sum S = sum A^2 over the patch).
 *   4. centred focal coordinate c(u) = u for u < F/2, u - F otherwise (one unit = a tilt of
 *      2 pi / F radians per pupil pixel).
 *   5. flux = sum S;  mx = sum c(u) S over u != F/2,  my = sum c(v) S over v != F/2 (the Nyquist
 *      sample has no mirror partner and is left out of the first moments).
 *   6. a sub-aperture is valid iff sum A^2 >= 0.5 p^2; slopes sx = mx / flux, sy = my / flux
 *      there (in focal samples), 0 where invalid or flux == 0.
 *   7. optional detector image: the centred spot (index U = c(u) + F/2) summed over bs x bs
 *      blocks, n_pix = F / bs pixels across.
 *
 * The line DFT is the direct O(n^2) sum with a table of exp(-2 pi i j / F) (each entry from a
 * direct sin/cos call, index (u x) mod F reduced in integers); rows first, then columns.
 * Pins: tests/test_sh_oracle_pins.py.  Build: gcc -O2 -fPIC -shared -o libshoracle.so sh_oracle.c -lm
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

/* out[u] = sum_{x<n} in[x] w[(u x) mod n], u < n: the plain n-point DFT of the (zero-padded) line. */
static void dft_line(int n, const double *w, const double *in, double *out)
{
    for (int u = 0; u < n; ++u) {
        double sr = 0.0, si = 0.0;
        int m = 0;
        for (int x = 0; x < n; ++x) {
            const double c = w[2 * m], s = w[2 * m + 1];
            sr += in[2 * x] * c - in[2 * x + 1] * s;
            si += in[2 * x] * s + in[2 * x + 1] * c;
            m += u;
            if (m >= n) m -= n;
        }
        out[2 * u] = sr;
        out[2 * u + 1] = si;
    }
}

/* Steps 2-3 for one patch: e [p][p][2] -> S [F][F]. */
void sho_spot(int p, int F, const double *e, double *S)
{
    double *w = (double *)malloc(sizeof(double) * 2 * (size_t)F);
    double *T = (double *)calloc((size_t)F * F * 2, sizeof(double));   /* [y][u], rows y >= p stay zero */
    double *col = (double *)malloc(sizeof(double) * 2 * (size_t)F);
    double *tmp = (double *)malloc(sizeof(double) * 2 * (size_t)F);
    double *row = (double *)calloc((size_t)F * 2, sizeof(double));     /* one zero-padded patch row */
    for (int j = 0; j < F; ++j) {
        const double a = -2.0 * M_PI * (double)j / (double)F;
        w[2 * j] = cos(a);
        w[2 * j + 1] = sin(a);
    }
    for (int y = 0; y < p; ++y) {
        memcpy(row, e + 2 * (size_t)y * p, sizeof(double) * 2 * (size_t)p);     /* samples p..F-1 stay zero */
        dft_line(F, w, row, T + 2 * (size_t)y * F);
    }
    const double inv = 1.0 / ((double)F * (double)F);
    for (int u = 0; u < F; ++u) {
        for (int y = 0; y < F; ++y) {
            col[2 * y] = T[2 * ((size_t)y * F + u)];
            col[2 * y + 1] = T[2 * ((size_t)y * F + u) + 1];
        }
        dft_line(F, w, col, tmp);
        for (int v = 0; v < F; ++v)
            S[(size_t)v * F + u] = (tmp[2 * v] * tmp[2 * v] + tmp[2 * v + 1] * tmp[2 * v + 1]) * inv;
    }
    free(w); free(T); free(col); free(tmp); free(row);
}

static int cfreq(int u, int F) { return u < F / 2 ? u : u - F; }

/*
 * The whole path.  amp, phase: float32 [B][P][P] (converted to double here).
 *   slopes : [B][2][n_sub][n_sub] (plane 0 = sx, 1 = sy), focal samples
 *   flux   : NULL or [B][n_sub][n_sub]
 *   spots  : NULL or [B][n_sub][n_sub][n_pix][n_pix], n_pix = F / bs
 * Returns 0, 1 on bad arguments, 3 out of memory.
 */
int sh_oracle_compute(int P, int n_sub, int F, int bs, int B, const float *amp, const float *phase,
                      double *slopes, double *flux, double *spots)
{
    if (P < 1 || n_sub < 1 || P % n_sub != 0 || F < 2 || (F & 1) || bs < 1 || F % bs != 0 || B < 1 ||
        !amp || !phase || !slopes)
        return 1;
    const int p = P / n_sub, npix = F / bs;
    if (p > F) return 1;
    double *e = (double *)malloc(sizeof(double) * 2 * (size_t)p * p);
    double *S = (double *)malloc(sizeof(double) * (size_t)F * F);
    if (!e || !S) { free(e); free(S); return 3; }
    for (int b = 0; b < B; ++b)
        for (int sy = 0; sy < n_sub; ++sy)
            for (int sx = 0; sx < n_sub; ++sx) {
                double a2 = 0.0;
                for (int y = 0; y < p; ++y)
                    for (int x = 0; x < p; ++x) {
                        const size_t idx = ((size_t)b * P + (size_t)sy * p + y) * P + (size_t)sx * p + x;
                        const double A = (double)amp[idx], ph = (double)phase[idx];
                        e[2 * ((size_t)y * p + x)] = A * cos(ph);
                        e[2 * ((size_t)y * p + x) + 1] = A * sin(ph);
                        a2 += A * A;
                    }
                sho_spot(p, F, e, S);
                double fl = 0.0, mx = 0.0, my = 0.0;
                for (int v = 0; v < F; ++v)
                    for (int u = 0; u < F; ++u) {
                        const double s = S[(size_t)v * F + u];
                        fl += s;
                        if (u != F / 2) mx += (double)cfreq(u, F) * s;
                        if (v != F / 2) my += (double)cfreq(v, F) * s;
                    }
                const size_t sub = ((size_t)b * n_sub + sy) * n_sub + sx;
                const int valid = a2 >= 0.5 * (double)p * (double)p && fl > 0.0;
                slopes[((size_t)b * 2 + 0) * n_sub * n_sub + (size_t)sy * n_sub + sx] = valid ? mx / fl : 0.0;
                slopes[((size_t)b * 2 + 1) * n_sub * n_sub + (size_t)sy * n_sub + sx] = valid ? my / fl : 0.0;
                if (flux) flux[sub] = fl;
                if (spots) {
                    double *px = spots + sub * (size_t)npix * npix;
                    memset(px, 0, sizeof(double) * (size_t)npix * npix);
                    for (int v = 0; v < F; ++v)
                        for (int u = 0; u < F; ++u) {
                            const int V = cfreq(v, F) + F / 2, U = cfreq(u, F) + F / 2;
                            px[(size_t)(V / bs) * npix + U / bs] += S[(size_t)v * F + u];
                        }
                }
            }
    free(e); free(S);
    return 0;
}
