// sh.cu -- Shack-Hartmann spots and centroids (include/sh.h).
//
// One CTA per sub-aperture; patch, row spectra and twiddle table in shared memory.  The patch is
// p x p (p <= 32) inside an F x F padded array, so the row pass is a SKINNY contraction,
//   T[y][u] = sum_{x<p} e[y][x] w^(u x)        (p x F values, p terms each),   w = exp(-2 pi i / F),
// never an FFT over mostly-zero data.  The column pass f[v][u] = sum_{y<p} T[y][u] w^(v y) has two forms:
//   k_shp<8>, k_shp<16> : p = 8 or 16 and bs | F/p -- F/p twisted p-point DFTs per column (p - 1 complex
//                         multiplies + one radix-p butterfly per p samples), the fast path;
//   k_sh<RV, CU>        : any other p or binning -- the direct contraction, RV x CU samples per lane.
// Pixel sums, flux and first moments accumulate in registers and are reduced by shuffles in a fixed
// order: deterministic, no atomics.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <new>

#include "../../include/sh.h"
#include "pyr_fft.cuh"   // packed FP32x2 complex helpers and the radix-8 butterfly

namespace {

constexpr int SH_THREADS = 128;

struct ShDev {
    int P, ns, p, F, bs, npix, B;
};

// RV x CU = rows x columns (32 apart) of the spot a lane evaluates together: CU loads of T and RV
// twiddle broadcasts feed RV * CU complex FMAs, which keeps the FMA pipe, not shared memory, the
// limiter (RV = 8, CU = 2: 12 wavefronts per 64 FFMA instructions).  bs % RV == 0, F % (32 CU) == 0
// or CU == 1.
template <int RV, int CU>
__global__ void __launch_bounds__(SH_THREADS)
k_sh(const ShDev d, const float *__restrict__ amp, const float *__restrict__ phase, float *__restrict__ slopes,
     float *__restrict__ flux, float *__restrict__ spots) {
    extern __shared__ float2 sm[];
    const int p = d.p, F = d.F, bs = d.bs, npix = d.npix, tid = threadIdx.x;
    const int warp = tid >> 5, lane = tid & 31;
    constexpr int NW = SH_THREADS / 32;
    float2 *w = sm;                 // [F]     exp(-2 pi i j / F)
    float2 *e = w + F;              // [p][p]  A exp(i phi)
    float2 *T = e + p * p;          // [p][F]
    __shared__ float red[4][NW];
    const int sub = blockIdx.x;     // (b, sy, sx)
    const int sx = sub % d.ns, sy = (sub / d.ns) % d.ns, b = sub / (d.ns * d.ns);

    for (int j = tid; j < F; j += SH_THREADS) {
        float s, c;
        sincospif(-2.0f * (float)j / (float)F, &s, &c);
        w[j] = make_float2(c, s);
    }
    float a2 = 0.f;
    for (int i = tid; i < p * p; i += SH_THREADS) {
        const int y = i / p, x = i % p;
        const size_t idx = ((size_t)b * d.P + (size_t)sy * p + y) * d.P + (size_t)sx * p + x;
        const float A = __ldg(&amp[idx]);
        float s, c;
        sincosf(__ldg(&phase[idx]), &s, &c);
        e[i] = make_float2(A * c, A * s);
        a2 += A * A;
    }
    __syncthreads();
    // rows: T[y][u], u natural; lanes take consecutive u (conflict-free), e[y][x] is a broadcast
    for (int i = tid; i < p * F; i += SH_THREADS) {
        const int y = i / F, u = i % F;
        float tr = 0.f, ti = 0.f;
        int m = 0;
        for (int x = 0; x < p; ++x) {
            const float2 ev = e[y * p + x], ww = w[m];
            tr = fmaf(ev.x, ww.x, fmaf(-ev.y, ww.y, tr));
            ti = fmaf(ev.x, ww.y, fmaf(ev.y, ww.x, ti));
            m = (m + u) & (F - 1);
        }
        T[i] = make_float2(tr, ti);
    }
    __syncthreads();
    // columns, modulus, moments.  A warp owns the band of bs rows of one detector-pixel row; its lanes
    // take 32 consecutive centred columns U (consecutive u: conflict-free loads of T, the twiddle of
    // a row is a broadcast) and RV rows at a time; pixel sums by a segmented shuffle reduction.
    const float inv = 1.0f / ((float)F * (float)F);
    float fl = 0.f, mx = 0.f, my = 0.f;
    float *px = spots ? spots + (size_t)sub * npix * npix : nullptr;
    for (int Y = warp; Y < npix; Y += NW) {
        float wide = 0.f;                       // pixel sum across chunks when bs > 32
        for (int j0 = 0; j0 < F; j0 += 32 * CU) {
            int cu[CU], u[CU];
            bool on[CU];
            float colsum[CU];
#pragma unroll
            for (int c = 0; c < CU; ++c) {
                const int U = j0 + 32 * c + lane;
                cu[c] = U - F / 2;
                u[c] = cu[c] & (F - 1);
                on[c] = U < F;
                colsum[c] = 0.f;
            }
            for (int dv0 = 0; dv0 < bs; dv0 += RV) {
                float fr[RV][CU], fi[RV][CU];
                int m[RV], v[RV], cv[RV];
#pragma unroll
                for (int r = 0; r < RV; ++r) {
                    cv[r] = Y * bs + dv0 + r - F / 2;
                    v[r] = cv[r] & (F - 1);
                    m[r] = 0;
#pragma unroll
                    for (int c = 0; c < CU; ++c) fr[r][c] = fi[r][c] = 0.f;
                }
                for (int y = 0; y < p; ++y) {
                    float2 t[CU];
#pragma unroll
                    for (int c = 0; c < CU; ++c) t[c] = T[y * F + u[c]];
#pragma unroll
                    for (int r = 0; r < RV; ++r) {
                        const float2 ww = w[m[r]];
#pragma unroll
                        for (int c = 0; c < CU; ++c) {
                            fr[r][c] = fmaf(t[c].x, ww.x, fmaf(-t[c].y, ww.y, fr[r][c]));
                            fi[r][c] = fmaf(t[c].x, ww.y, fmaf(t[c].y, ww.x, fi[r][c]));
                        }
                        m[r] = (m[r] + v[r]) & (F - 1);
                    }
                }
#pragma unroll
                for (int r = 0; r < RV; ++r)
#pragma unroll
                    for (int c = 0; c < CU; ++c) {
                        const float s = on[c] ? (fr[r][c] * fr[r][c] + fi[r][c] * fi[r][c]) * inv : 0.f;
                        colsum[c] += s;
                        if (cu[c] != -F / 2) mx = fmaf((float)cu[c], s, mx);
                        if (cv[r] != -F / 2) my = fmaf((float)cv[r], s, my);
                    }
            }
#pragma unroll
            for (int c = 0; c < CU; ++c) {
                fl += colsum[c];
                if (px) {
                    const int U = j0 + 32 * c + lane;
                    float a = colsum[c];
                    if (bs <= 32) {
                        for (int o = 1; o < bs; o <<= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
                        if (on[c] && (U % bs) == 0) px[Y * npix + U / bs] = a;
                    } else {
#pragma unroll
                        for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
                        wide += a;
                        if ((j0 + 32 * c + 32) % bs == 0) {
                            if (lane == 0) px[Y * npix + (j0 + 32 * c) / bs] = wide;
                            wide = 0.f;
                        }
                    }
                }
            }
        }
    }
    // block reduction in a fixed order: lanes by shuffle, then the warps one after the other
    float vals[4] = {fl, mx, my, a2};
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        float v = vals[k];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if (lane == 0) red[k][warp] = v;
    }
    __syncthreads();
    if (tid == 0) {
        float r[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            r[k] = 0.f;
            for (int wi = 0; wi < NW; ++wi) r[k] += red[k][wi];
        }
        const bool valid = r[3] >= 0.5f * (float)(p * p) && r[0] > 0.f;
        const int n2 = d.ns * d.ns;
        slopes[((size_t)b * 2 + 0) * n2 + sy * d.ns + sx] = valid ? r[1] / r[0] : 0.f;
        slopes[((size_t)b * 2 + 1) * n2 + sy * d.ns + sx] = valid ? r[2] / r[0] : 0.f;
        if (flux) flux[sub] = r[0];
    }
}

// ---------------------------------------------------------------- p = 8 or 16: pruned column transform
// With PP non-zero rows the F-point column transform splits exactly into F/PP twisted PP-point DFTs:
//     f[(F/PP) a + b][u] = sum_{y<PP} ( T[y][u] w^(b y) ) exp(-2 pi i a y / PP),      a < PP, b < F/PP,
// i.e. PP - 1 complex multiplies and one radix-PP butterfly (pyr_fft.cuh) per PP spot samples instead of
// PP^2 complex FMAs -- about a third of the instructions of k_sh at PP = 8.  A lane keeps the PP values T[.][u] of its
// column in registers and walks b; the PP samples of a task lie in PP different detector-pixel rows
// (centred row V = (F/PP) a' + b, a' = (a + PP/2) mod PP), so with bs | F/PP a block of bs consecutive b
// feeds exactly one pixel row per a': PP running pixel sums per lane, reduced over bs lanes by shuffles.
// Requires p == PP and bs | F/PP (bs <= 32); everything else falls back to k_sh.
template <int PP>
__global__ void __launch_bounds__(SH_THREADS)
k_shp(const ShDev d, const float *__restrict__ amp, const float *__restrict__ phase, float *__restrict__ slopes,
      float *__restrict__ flux, float *__restrict__ spots) {
    using pyr::cmul;
    extern __shared__ float2 sm[];
    constexpr int p = PP;
    const int F = d.F, bs = d.bs, npix = d.npix, tid = threadIdx.x;
    const int warp = tid >> 5, lane = tid & 31, Q = F / PP;
    constexpr int NW = SH_THREADS / 32;
    float2 *w = sm;                 // [F]     exp(-2 pi i j / F)
    float2 *e = w + F;              // [PP][PP]  A exp(i phi)
    float2 *T = e + p * p;          // [PP][F]
    __shared__ float red[4][NW];
    const int sub = blockIdx.x;
    const int sx = sub % d.ns, sy = (sub / d.ns) % d.ns, b_ = sub / (d.ns * d.ns);

    for (int j = tid; j < F; j += SH_THREADS) {
        float s, c;
        sincospif(-2.0f * (float)j / (float)F, &s, &c);
        w[j] = make_float2(c, s);
    }
    float a2 = 0.f;
    for (int i = tid; i < p * p; i += SH_THREADS) {
        const int y = i / p, x = i % p;
        const size_t idx = ((size_t)b_ * d.P + (size_t)sy * p + y) * d.P + (size_t)sx * p + x;
        const float A = __ldg(&amp[idx]);
        float s, c;
        sincosf(__ldg(&phase[idx]), &s, &c);
        e[i] = make_float2(A * c, A * s);
        a2 += A * A;
    }
    __syncthreads();
    for (int i = tid; i < p * F; i += SH_THREADS) {       // rows: T[y][u]
        const int y = i / F, u = i % F;
        float2 t = make_float2(0.f, 0.f);
        int m = 0;
#pragma unroll
        for (int x = 0; x < p; ++x) {
            t = pyr::cadd(t, cmul(e[y * p + x], w[m]));
            m = (m + u) & (F - 1);
        }
        T[i] = t;
    }
    __syncthreads();
    const float inv = 1.0f / ((float)F * (float)F);
    float fl = 0.f, mx = 0.f, my = 0.f;
    float *px = spots ? spots + (size_t)sub * npix * npix : nullptr;
    const int nblk = Q / bs, nchunk = (F + 31) / 32;
    for (int job = warp; job < nblk * nchunk; job += NW) {
        const int blk = job / nchunk, j0 = (job % nchunk) * 32;
        const int U = j0 + lane, cu = U - F / 2, u = cu & (F - 1);
        const bool on = U < F;
        // (lanes beyond F hold zeros: no selects in the loop.  The loop is issue-bound with a busy ALU
        // pipe, so the twiddles w^(bb y) are powers of one loaded value and the row coordinates are
        // floats advanced by 1 per step, not integer index arithmetic and conversions.)
        float2 t[PP];
#pragma unroll
        for (int y = 0; y < PP; ++y) t[y] = on ? T[y * F + u] : make_float2(0.f, 0.f);
        float pacc[PP], cvf[PP];
#pragma unroll
        for (int a = 0; a < PP; ++a) {
            pacc[a] = 0.f;
            cvf[a] = (float)(Q * ((a + PP / 2) % PP) + blk * bs - F / 2);   // centred row of output a at db = 0
        }
        const float cuf = cu != -F / 2 ? (float)cu : 0.f;               // Nyquist column: no first moment
        for (int db = 0; db < bs; ++db) {
            const int bb = blk * bs + db;
            float2 v[PP], o = w[bb];
            const float2 o1 = o;
            v[0] = t[0];
#pragma unroll
            for (int y = 1; y < PP; ++y) {                      // o = w^(bb y)
                v[y] = cmul(t[y], o);
                if (y + 1 < PP) o = cmul(o, o1);
            }
            pyr::dftR<PP, -1>(v);                               // v[a] = f[Q a + bb][u]
            float srow = 0.f;
#pragma unroll
            for (int a = 0; a < PP; ++a) {
                const float s = (v[a].x * v[a].x + v[a].y * v[a].y) * inv;
                pacc[(a + PP / 2) % PP] += s;
                srow += s;
                my = fmaf(cvf[a], s, my);
                cvf[a] += 1.0f;
            }
            if (bb == 0) {                                      // a = PP/2 is the Nyquist row cv = -F/2: take it back
                const float sn = (v[PP / 2].x * v[PP / 2].x + v[PP / 2].y * v[PP / 2].y) * inv;
                my = fmaf((float)(F / 2), sn, my);
            }
            fl += srow;
            mx = fmaf(cuf, srow, mx);
        }
        if (px) {
#pragma unroll
            for (int ap = 0; ap < PP; ++ap) {
                float a = pacc[ap];
                for (int o = 1; o < bs; o <<= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
                if (on && (U % bs) == 0) px[((Q * ap + blk * bs) / bs) * npix + U / bs] = a;
            }
        }
    }
    float vals[4] = {fl, mx, my, a2};
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        float v = vals[k];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if (lane == 0) red[k][warp] = v;
    }
    __syncthreads();
    if (tid == 0) {
        float r[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            r[k] = 0.f;
            for (int wi = 0; wi < NW; ++wi) r[k] += red[k][wi];
        }
        const bool valid = r[3] >= 0.5f * (float)(p * p) && r[0] > 0.f;
        const int n2 = d.ns * d.ns;
        slopes[((size_t)b_ * 2 + 0) * n2 + sy * d.ns + sx] = valid ? r[1] / r[0] : 0.f;
        slopes[((size_t)b_ * 2 + 1) * n2 + sy * d.ns + sx] = valid ? r[2] / r[0] : 0.f;
        if (flux) flux[sub] = r[0];
    }
}

typedef void (*sh_kernel_t)(const ShDev, const float *, const float *, float *, float *, float *);

thread_local int g_err = 0;
thread_local char g_msg[256] = "";

int set_err(int code, const char *fmt, ...) {
    g_err = code;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_msg, sizeof(g_msg), fmt, ap);
    va_end(ap);
    return code;
}

}  // namespace

struct sh_plan {
    ShDev d;
    size_t smem;
    sh_kernel_t kernel;
};

extern "C" {

int sh_last_error(void) { return g_err; }
const char *sh_last_error_string(void) { return g_msg; }

sh_plan *sh_plan_create(int P, int ns, int F, int bs, int B) {
    if (P < 1 || ns < 1 || P % ns != 0) { set_err(1, "n_sub=%d must divide N_pup=%d", ns, P); return nullptr; }
    const int p = P / ns;
    if (p > 32) { set_err(2, "sub-aperture of %d pixels: at most 32 supported", p); return nullptr; }
    if (F < 8 || F > 256 || (F & (F - 1)) || F < p) { set_err(1, "F=%d must be a power of two in [max(p, 8), 256]", F); return nullptr; }
    if (bs < 1 || F % bs != 0) { set_err(1, "spot_binning=%d must divide F", bs); return nullptr; }
    if (B < 1) { set_err(1, "batch=%d must be >= 1", B); return nullptr; }
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { set_err(4, "no CUDA device: %s", cudaGetErrorString(cudaGetLastError())); return nullptr; }
    sh_plan *pl = new (std::nothrow) sh_plan();
    if (!pl) { set_err(3, "host allocation failed"); return nullptr; }
    pl->d = ShDev{P, ns, p, F, bs, F / bs, B};
    pl->smem = (size_t)(F + p * p + p * F) * sizeof(float2);
    if (p == 8 && (F / 8) % bs == 0 && bs <= 32) pl->kernel = k_shp<8>;
    else if (p == 16 && F >= 32 && (F / 16) % bs == 0 && bs <= 32) pl->kernel = k_shp<16>;
    else if (F >= 128 && bs % 4 == 0) pl->kernel = k_sh<4, 4>;
    else if (F >= 64) pl->kernel = bs % 8 == 0 ? k_sh<8, 2> : bs % 4 == 0 ? k_sh<4, 2> : bs % 2 == 0 ? k_sh<2, 2> : k_sh<1, 2>;
    else pl->kernel = bs % 4 == 0 ? k_sh<4, 1> : bs % 2 == 0 ? k_sh<2, 1> : k_sh<1, 1>;
    cudaError_t e = cudaFuncSetAttribute((const void *)pl->kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl->smem);
    if (e != cudaSuccess) {
        set_err(4, "kernel setup failed: %s", cudaGetErrorString(e));
        delete pl;
        return nullptr;
    }
    return pl;
}

int sh_compute(sh_plan *pl, const float *amp, const float *phase, float *out_slopes, float *out_flux,
               float *out_spots, void *stream) {
    if (!pl || !amp || !phase || !out_slopes) return set_err(1, "sh_compute: NULL plan, amp, phase or out_slopes");
    const ShDev &d = pl->d;
    pl->kernel<<<d.B * d.ns * d.ns, SH_THREADS, pl->smem, (cudaStream_t)stream>>>(d, amp, phase, out_slopes, out_flux, out_spots);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return set_err(4, "sh_compute: launch failed: %s", cudaGetErrorString(e));
    return 0;
}

void sh_plan_destroy(sh_plan *pl) { delete pl; }

}  // extern "C"
