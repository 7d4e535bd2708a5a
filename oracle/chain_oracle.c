/*
 * chain_oracle.c -- CPU oracle for the steps either side of the wavefront sensor.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/ and bench.py's cpu legs may build, load or
 * call it.  It shares no source, header, table or helper with the CUDA library (libpyr).
 *
 * The paper names these processing objects and their parameters but prints no formula for any of them
 * (Table 4, PAPER.md:311-315 atmosphere / propagation, 323 `CCD`, 327 `PyrSlopec`, 332 `Modalrec`, 337
 * `PyrPupdataCalibrator`; Listing 2).  What is written out here, step by step,
 * is the reading listed in DESIGN.md section 14 (readings A1-A4, C1-C7, U1, M1):
 *
 *   atmo   (AtmoEvolution + AtmoPropagation, finite periodic screens, geometric propagation):
 *          phase[b][y][x] = sum_l w_l bilerp(screen_l, y + dy[b][l], x + dx[b][l]), bilinear interpolation
 *          on the periodic S x S screen, double precision.
 *   ccd    (CCD): expected photo-electrons acc += gain * D over n_int steps, then photon noise (Poisson:
 *          inversion by sequential search below 30 e-, rounded normal approximation above), readout
 *          noise (normal), ADC (divide, round, clamp).  Random numbers: Philox4x32-10 (Salmon et al.,
 *          SC'11), counter = (pixel index, frame index, 0, 0), key = seed.  Every floating-point step of
 *          this model that decides an integer is taken in float32 with IEEE-exact operations only
 *          (add, multiply, fma, divide, sqrt, rint; exp / log / cos are polynomials of those, written out
 *          below), the precision the kernel computes in, so the CUDA path reproduces it bit for bit.
 *   pupdata (PyrPupdataCalibrator): valid iff the four-quadrant sum of a reference frame >= thr * its maximum.
 *   modalrec (Modalrec): modes = R . [sx at the valid pixels, sy at the valid pixels], double precision.
 *   (PyrSlopec on detector pixels is pyro_slopes of pyr_oracle.c applied to the CCD frame.)
 *
 * Pins: tests/test_chain_oracle_pins.py (published Philox known-answer vectors, closed forms, brute force,
 * distribution moments, scipy's Poisson quantiles, library cross-checks).
 * Build: gcc -O2 -ffp-contract=off -fPIC -shared -o libchainoracle.so chain_oracle.c -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------------------------------------------ atmosphere (readings A1-A4) */

/* Bilinear interpolation of the periodic S x S screen at real coordinates (Y, X):
 * i = floor(Y), fy = Y - i (likewise j, fx), indices wrapped mod S. */
static double bilerp_periodic(int S, const float *scr, double Y, double X)
{
    const double fyf = floor(Y), fxf = floor(X);
    const double fy = Y - fyf, fx = X - fxf;
    long long i = (long long)fyf % S, j = (long long)fxf % S;
    if (i < 0) i += S;
    if (j < 0) j += S;
    const long long i1 = (i + 1) % S, j1 = (j + 1) % S;
    const double s00 = scr[i * S + j], s01 = scr[i * S + j1], s10 = scr[i1 * S + j], s11 = scr[i1 * S + j1];
    return (1.0 - fy) * ((1.0 - fx) * s00 + fx * s01) + fy * ((1.0 - fx) * s10 + fx * s11);
}

/* phase[b][y][x] = sum_l weights[l] * bilerp(screens[l], y + shift[b][l][0], x + shift[b][l][1]).
 * screens: float32 [L][S][S]; weights: [L] or NULL (= 1); shift_yx: [B][L][2] pixels; out: [B][P][P]. */
int chain_oracle_atmo(int L, int S, int P, int B, const float *screens, const double *weights,
                      const double *shift_yx, double *out)
{
    if (L < 1 || S < 2 || P < 1 || B < 1 || !screens || !shift_yx || !out) return 1;
    for (int b = 0; b < B; ++b)
        for (int y = 0; y < P; ++y)
            for (int x = 0; x < P; ++x) {
                double acc = 0.0;
                for (int l = 0; l < L; ++l) {
                    const double dy = shift_yx[((size_t)b * L + l) * 2], dx = shift_yx[((size_t)b * L + l) * 2 + 1];
                    const double w = weights ? weights[l] : 1.0;
                    acc += w * bilerp_periodic(S, screens + (size_t)l * S * S, (double)y + dy, (double)x + dx);
                }
                out[((size_t)b * P + y) * P + x] = acc;
            }
    return 0;
}

/* ------------------------------------------------------------------ Philox4x32-10 (reading C4) */

/* Salmon, Moraes, Dror, Shaw, "Parallel random numbers: as easy as 1, 2, 3", SC'11: ten rounds of
 *   (c0, c1, c2, c3) <- (hi(M1 c2) ^ c1 ^ k0, lo(M1 c2), hi(M0 c0) ^ c3 ^ k1, lo(M0 c0)),
 * the key bumped by the Weyl constants (W0, W1) before every round but the first. */
void cho_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        if (r) { k0 += W0; k1 += W1; }
        const uint64_t p0 = (uint64_t)M0 * c0, p1 = (uint64_t)M1 * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* ------------------------------------------------------------------ float32 helpers of the noise model (reading C5)
 * IEEE-exact operations only, in a fixed order; compiled with -ffp-contract=off so that every fma is the one
 * written.  These define the generator's maps; their accuracy (about 1e-7 relative) is pinned against libm. */

static float bits_to_float(uint32_t b) { float f; memcpy(&f, &b, 4); return f; }
static uint32_t float_to_bits(float f) { uint32_t b; memcpy(&b, &f, 4); return b; }

/* uniform in (0, 1): the top 23 bits, centred in their cell, (k + 1/2) 2^-23 -- exact in float32, never 0 or 1 */
float cho_u01(uint32_t x) { return ((float)(x >> 9) + 0.5f) * 1.1920928955078125e-7f; }

/* exp(-lam), 0 <= lam <= 80: k = rint(-lam log2 e), r = -lam - k ln 2 (two-step), degree-6 polynomial, scale 2^k */
float cho_exp_neg(float lam)
{
    const float x = -lam;
    const float k = rintf(x * 1.44269504088896341f);
    float r = fmaf(k, -0.693359375f, x);
    r = fmaf(k, 2.12194440e-4f, r);
    float p = 1.9875691500e-4f;
    p = fmaf(p, r, 1.3981999507e-3f);
    p = fmaf(p, r, 8.3334519073e-3f);
    p = fmaf(p, r, 4.1665795894e-2f);
    p = fmaf(p, r, 1.6666665459e-1f);
    p = fmaf(p, r, 5.0000001201e-1f);
    const float r2 = r * r;
    float y = fmaf(p, r2, r);
    y = y + 1.0f;
    return y * bits_to_float((uint32_t)((int)k + 127) << 23);
}

/* log(u), u a normal float in (0, 1]: u = m 2^e with m in [sqrt(1/2), sqrt 2), polynomial in m - 1 */
float cho_log(float u)
{
    const uint32_t b = float_to_bits(u);
    int e = (int)((b >> 23) & 0xffu) - 126;
    float x = bits_to_float((b & 0x007fffffu) | 0x3f000000u);        /* in [0.5, 1) */
    if (x < 0.707106781186547524f) { e -= 1; x = (x + x) - 1.0f; } else { x = x - 1.0f; }
    const float z = x * x;
    float y = 7.0376836292e-2f;
    y = fmaf(y, x, -1.1514610310e-1f);
    y = fmaf(y, x, 1.1676998740e-1f);
    y = fmaf(y, x, -1.2420140846e-1f);
    y = fmaf(y, x, 1.4249322787e-1f);
    y = fmaf(y, x, -1.6668057665e-1f);
    y = fmaf(y, x, 2.0000714765e-1f);
    y = fmaf(y, x, -2.4999993993e-1f);
    y = fmaf(y, x, 3.3333331174e-1f);
    y = (y * x) * z;
    const float fe = (float)e;
    y = fmaf(fe, -2.12194440e-4f, y);
    y = fmaf(-0.5f, z, y);
    float r = x + y;
    r = fmaf(fe, 0.693359375f, r);
    return r;
}

/* cos(2 pi u), u in [0, 1): octant j = floor(8u), f = 8u - j, reduced angle a = f pi/4 (even j) or (1 - f) pi/4 */
float cho_cos2pi(float u)
{
    const float t = u * 8.0f;
    const int j = (int)t;
    const float f = t - (float)j;
    const float a = ((j & 1) ? (1.0f - f) : f) * 0.78539816339744830962f;
    const float z = a * a;
    float s = -1.9515295891e-4f;
    s = fmaf(s, z, 8.3321608736e-3f);
    s = fmaf(s, z, -1.6666654611e-1f);
    s = fmaf(s * z, a, a);                                          /* sin a */
    float c = 2.443315711809948e-5f;
    c = fmaf(c, z, -1.388731625493765e-3f);
    c = fmaf(c, z, 4.166664568298827e-2f);
    c = fmaf(c, z * z, fmaf(-0.5f, z, 1.0f));                       /* cos a */
    switch (j & 7) {
        case 0: return c;
        case 1: return s;
        case 2: return -s;
        case 3: return -c;
        case 4: return -c;
        case 5: return -s;
        case 6: return s;
        default: return c;
    }
}

/* standard normal deviate from two uniforms (Box-Muller, cosine branch) */
float cho_normal(float ua, float ub)
{
    const float m = sqrtf(-2.0f * cho_log(ua));
    return m * cho_cos2pi(ub);
}

/* Poisson deviate with mean lam >= 0 as a float count.  lam < 30: inversion by sequential search,
 * p_0 = exp(-lam), p_n = p_{n-1} lam / n, the smallest n with ua <= p_0 + ... + p_n (at most 200);
 * otherwise the rounded normal approximation max(0, rint(lam + sqrt(lam) z)). */
float cho_poisson(float lam, float ua, float ub)
{
    if (!(lam > 0.0f)) return 0.0f;
    if (lam < 30.0f) {
        float p = cho_exp_neg(lam), s = p;
        int n = 0;
        while (ua > s && n < 200) {
            ++n;
            p = (p * lam) / (float)n;
            s = s + p;
        }
        return (float)n;
    }
    const float v = fmaf(sqrtf(lam), cho_normal(ua, ub), lam);
    const float n = rintf(v);
    return n > 0.0f ? n : 0.0f;
}

/* ------------------------------------------------------------------ CCD (readings C1-C7)
 * One call = one simulation step.  acc[i] = fma(gain, D[i], acc[i]) (float32).  When `readout` is non-zero the
 * frame is produced from acc and acc is cleared:
 *   e = acc;  photon noise: e = Poisson(e) with (ua, ub) = u01 of Philox words 0, 1;
 *   readout noise: e = fma(sigma, normal(u01(word 2), u01(word 3)), e);
 *   adu_gain > 0: pixel = min(max(rint(e / adu_gain), 0), 2^n_bits - 1), else pixel = e.
 * Philox counter = (i, frame_index, 0, 0) with i the linear pixel index in [B][Nd][Nd], key = (seed lo, seed hi). */
int chain_oracle_ccd(long long n, float *acc, const float *D, float gain, int readout, int photon_noise,
                     int readout_noise, float sigma, float adu_gain, int n_bits, uint64_t seed,
                     uint32_t frame_index, float *pixels)
{
    if (n < 1 || !acc || !D || (readout && !pixels)) return 1;
    const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    const float full = (float)((1u << (n_bits > 0 && n_bits < 31 ? n_bits : 16)) - 1u);
    for (long long i = 0; i < n; ++i) {
        acc[i] = fmaf(gain, D[i], acc[i]);
        if (!readout) continue;
        float e = acc[i];
        acc[i] = 0.0f;
        if (photon_noise || readout_noise) {
            const uint32_t ctr[4] = {(uint32_t)i, frame_index, 0u, 0u};
            uint32_t w[4];
            cho_philox4x32_10(ctr, key, w);
            if (photon_noise) e = cho_poisson(e, cho_u01(w[0]), cho_u01(w[1]));
            if (readout_noise) e = fmaf(sigma, cho_normal(cho_u01(w[2]), cho_u01(w[3])), e);
        }
        if (adu_gain > 0.0f) {
            float v = rintf(e / adu_gain);
            v = v > 0.0f ? v : 0.0f;
            e = v < full ? v : full;
        }
        pixels[i] = e;
    }
    return 0;
}

/* ------------------------------------------------------------------ PupData from a reference frame (reading U1)
 * T[Y][X] = (Qa + Qb) + (Qc + Qd) of the reference frame (float32, this order); valid iff T >= thr * max T
 * (one float32 multiply). */
int chain_oracle_pupdata(int Nd, const float *ref, float thr, unsigned char *valid)
{
    if (Nd < 2 || (Nd & 1) || !ref || !valid) return 1;
    const int Nq = Nd / 2;
    float tmax = 0.0f;
    for (int pass = 0; pass < 2; ++pass)
        for (int Y = 0; Y < Nq; ++Y)
            for (int X = 0; X < Nq; ++X) {
                const float Qa = ref[(size_t)Y * Nd + X], Qb = ref[(size_t)Y * Nd + X + Nq];
                const float Qc = ref[(size_t)(Y + Nq) * Nd + X], Qd = ref[(size_t)(Y + Nq) * Nd + X + Nq];
                const float T = (Qa + Qb) + (Qc + Qd);
                if (pass == 0) { if (T > tmax) tmax = T; }
                else valid[(size_t)Y * Nq + X] = (T >= thr * tmax) ? 1 : 0;
            }
    return 0;
}

/* ------------------------------------------------------------------ Modalrec (reading M1)
 * sv = [sx[Y][X] for valid (Y, X) in row-major order, then sy likewise]; modes[b][m] = sum_i R[m][i] sv[b][i].
 * slopes: float32 dense [B][2][Nq][Nq]; R: float32 [n_modes][2 n_valid]; out: double [B][n_modes]. */
int chain_oracle_modalrec(int n_modes, int Nq, int B, const unsigned char *valid, const float *R,
                          const float *slopes, double *modes)
{
    if (n_modes < 1 || Nq < 1 || B < 1 || !valid || !R || !slopes || !modes) return 1;
    const size_t nq2 = (size_t)Nq * Nq;
    size_t nv = 0;
    for (size_t i = 0; i < nq2; ++i) nv += valid[i] ? 1 : 0;
    double *sv = (double *)malloc(sizeof(double) * (2 * nv + 1));
    if (!sv) return 3;
    for (int b = 0; b < B; ++b) {
        size_t c = 0;
        for (int plane = 0; plane < 2; ++plane)
            for (size_t i = 0; i < nq2; ++i)
                if (valid[i]) sv[c++] = (double)slopes[((size_t)b * 2 + plane) * nq2 + i];
        for (int m = 0; m < n_modes; ++m) {
            double acc = 0.0;
            for (size_t i = 0; i < 2 * nv; ++i) acc += (double)R[(size_t)m * 2 * nv + i] * sv[i];
            modes[(size_t)b * n_modes + m] = acc;
        }
    }
    free(sv);
    return 0;
}
