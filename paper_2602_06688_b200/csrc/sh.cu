// sh.cu -- Shack-Hartmann spots and centroids (include/sh.h).
//
// One CTA per sub-aperture; patch, row spectra and twiddles in shared memory.  The patch is
// p x p (p <= 32) inside an F x F padded array, F any even number (the paper's 56, 68, 240 of Table 2,
// PAPER.md:194, 196-197, are not powers of two), so both passes are SKINNY:
//   rows     T[y][u] = sum_{x<p} e[y][x] w^(u x)        (p x F values),        w = exp(-2 pi i / F),
//   columns  f[v][u] = sum_{y<p} T[y][u] w^(v y)        (F x F values),
// never an FFT over mostly-zero data, and no power-of-two assumption anywhere (indices wrap by a conditional
// subtract; w comes from a table the plan builds once in double).  Two kernels:
//   k_shp<PP>, PP = 4, 8, 16 : p = PP, PP | F and bs | F/PP -- with PP non-zero inputs an F-point transform
//                         splits exactly into F/PP twisted PP-point DFTs (PP - 1 complex multiplies + one
//                         radix-PP butterfly per PP outputs); used for both passes, the fast path;
//   k_sh<RV, CU>        : any other p or binning -- the direct contractions, RV x CU samples per lane.
// Pixel sums, flux and first moments accumulate in registers / shared memory and are reduced in a fixed
// order: deterministic, no atomics.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <new>
#include <vector>

#include "../../include/sh.h"
#include "pyr_fft.cuh"   // packed FP32x2 complex helpers and the radix-4/8/16 butterflies

namespace {

constexpr int SH_THREADS = 128;
constexpr int NW = SH_THREADS / 32;

struct ShDev {
    int P, ns, p, F, bs, npix, B;
    const float2 *w;                // [F] exp(-2 pi i j / F)
};

// patch e = A exp(i phi) of sub-aperture (b, sy, sx) into shared memory; returns this thread's share of sum A^2
__device__ __forceinline__ float load_patch(const ShDev &d, const float *__restrict__ amp, const float *__restrict__ phase,
                                            int b, int sy, int sx, float2 *e) {
    const int p = d.p;
    float a2 = 0.f;
    for (int i = threadIdx.x; i < p * p; i += SH_THREADS) {
        const int y = i / p, x = i % p;
        const size_t idx = ((size_t)b * d.P + (size_t)sy * p + y) * d.P + (size_t)sx * p + x;
        const float A = __ldg(&amp[idx]);
        float s, c;
        sincosf(__ldg(&phase[idx]), &s, &c);
        e[i] = make_float2(A * c, A * s);
        a2 += A * A;
    }
    return a2;
}

// block reduction of (flux, mx, my, sum A^2) in a fixed order -- lanes by shuffle, then the warps one after
// the other -- and the slopes / flux of the sub-aperture (steps 5-6 of the definition).
__device__ __forceinline__ void finish(const ShDev &d, float fl, float mx, float my, float a2, float inv, int sub,
                                       float *__restrict__ slopes, float *__restrict__ flux, float (*red)[NW]) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float vals[4] = {fl, mx, my, a2};
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        float v = vals[k];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if (lane == 0) red[k][warp] = v;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        float r[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            r[k] = 0.f;
            for (int wi = 0; wi < NW; ++wi) r[k] += red[k][wi];
        }
        const int sx = sub % d.ns, sy = (sub / d.ns) % d.ns, b = sub / (d.ns * d.ns);
        const bool valid = r[3] >= 0.5f * (float)(d.p * d.p) && r[0] > 0.f;
        const int n2 = d.ns * d.ns;
        slopes[((size_t)b * 2 + 0) * n2 + sy * d.ns + sx] = valid ? r[1] / r[0] : 0.f;
        slopes[((size_t)b * 2 + 1) * n2 + sy * d.ns + sx] = valid ? r[2] / r[0] : 0.f;
        if (flux) flux[sub] = r[0] * inv;
    }
}

// ---------------------------------------------------------------- k_sh: direct contractions, any p <= 32, any even F
// RV x CU = rows x columns (32 apart) of the spot a lane evaluates together: CU loads of T and RV
// twiddle broadcasts feed RV * CU complex FMAs, which keeps the FMA pipe, not shared memory, the
// limiter.  bs % RV == 0.  A warp owns the band of bs rows of one detector-pixel row; its column sums go
// to a per-warp line of shared memory from which the pixels of that row are summed (any bs).
template <int RV, int CU>
__global__ void __launch_bounds__(SH_THREADS)
k_sh(const ShDev d, const float *__restrict__ amp, const float *__restrict__ phase, float *__restrict__ slopes,
     float *__restrict__ flux, float *__restrict__ spots) {
    extern __shared__ float2 sm[];
    const int p = d.p, F = d.F, bs = d.bs, npix = d.npix, tid = threadIdx.x;
    const int warp = tid >> 5, lane = tid & 31;
    float2 *w = sm;                 // [F]     exp(-2 pi i j / F)
    float2 *e = w + F;              // [p][p]  A exp(i phi)
    float2 *T = e + p * p;          // [p][F]
    float *rowbuf = reinterpret_cast<float *>(T + p * F) + warp * F;   // [NW][F] column sums of a pixel row
    __shared__ float red[4][NW];
    const int sub = blockIdx.x;     // (b, sy, sx)
    const int sx = sub % d.ns, sy = (sub / d.ns) % d.ns, b = sub / (d.ns * d.ns);

    for (int j = tid; j < F; j += SH_THREADS) w[j] = __ldg(&d.w[j]);
    const float a2 = load_patch(d, amp, phase, b, sy, sx, e);
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
            m += u;
            if (m >= F) m -= F;
        }
        T[i] = make_float2(tr, ti);
    }
    __syncthreads();
    // columns, modulus, moments.  Lanes take 32 consecutive centred columns U (consecutive u up to one wrap:
    // conflict-free loads of T, the twiddle of a row is a broadcast) and RV rows at a time.
    const float inv = 1.0f / ((float)F * (float)F);
    float fl = 0.f, mx = 0.f, my = 0.f;
    float *px = spots ? spots + (size_t)sub * npix * npix : nullptr;
    for (int Y = warp; Y < npix; Y += NW) {
        for (int j0 = 0; j0 < F; j0 += 32 * CU) {
            int cu[CU], u[CU];
            bool on[CU];
            float colsum[CU];
#pragma unroll
            for (int c = 0; c < CU; ++c) {
                const int U = j0 + 32 * c + lane;
                on[c] = U < F;
                cu[c] = U - F / 2;
                u[c] = on[c] ? (cu[c] < 0 ? cu[c] + F : cu[c]) : 0;
                colsum[c] = 0.f;
            }
            for (int dv0 = 0; dv0 < bs; dv0 += RV) {
                float fr[RV][CU], fi[RV][CU];
                int m[RV], v[RV], cv[RV];
#pragma unroll
                for (int r = 0; r < RV; ++r) {
                    cv[r] = Y * bs + dv0 + r - F / 2;
                    v[r] = cv[r] < 0 ? cv[r] + F : cv[r];
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
                        m[r] += v[r];
                        if (m[r] >= F) m[r] -= F;
                    }
                }
#pragma unroll
                for (int r = 0; r < RV; ++r)
#pragma unroll
                    for (int c = 0; c < CU; ++c) {
                        const float s = on[c] ? fr[r][c] * fr[r][c] + fi[r][c] * fi[r][c] : 0.f;
                        colsum[c] += s;
                        if (cu[c] != -F / 2) mx = fmaf((float)cu[c], s, mx);
                        if (cv[r] != -F / 2) my = fmaf((float)cv[r], s, my);
                    }
            }
#pragma unroll
            for (int c = 0; c < CU; ++c) {
                fl += colsum[c];
                if (px && on[c]) rowbuf[j0 + 32 * c + lane] = colsum[c];
            }
        }
        if (px) {
            __syncwarp();
            for (int X = lane; X < npix; X += 32) {
                float a = 0.f;
                for (int i = 0; i < bs; ++i) a += rowbuf[X * bs + i];
                px[Y * npix + X] = a * inv;
            }
            __syncwarp();
        }
    }
    finish(d, fl, mx, my, a2, inv, sub, slopes, flux, red);
}

// ---------------------------------------------------------------- k_shp: p = PP, PP | F: pruned transforms
// With PP non-zero inputs an F-point transform splits exactly into Q = F/PP twisted PP-point DFTs:
//     X[Q a + b] = sum_{n<PP} ( x[n] w^(b n) ) exp(-2 pi i a n / PP),      a < PP, b < Q,
// i.e. PP - 1 complex multiplies by tw[b][n] = w^(b n) and one radix-PP butterfly (pyr_fft.cuh) per PP outputs
// instead of PP^2 complex FMAs.  Rows: a thread takes one (y, b).  Columns: a lane keeps the PP values T[.][u] of
// its column in registers and walks b; the PP samples of a step lie in PP different detector-pixel rows
// (centred row V = Q a' + b, a' = (a + PP/2) mod PP), so with bs | Q a block of bs consecutive b feeds exactly
// one pixel row per a'.  Per step only sum |f|^2 is accumulated (packed, per a) plus the row sum weighted by
// its offset db inside the block; flux and both first moments follow from those at the end of the block
// (my = sum_a c0(a) Pa + sum_db db srow(db), mx = cu sum_a Pa), and everything is scaled by 1/F^2 once.
// Lanes cover CW = bs floor(32 / bs) consecutive columns, so a pixel never straddles two chunks; the pixel sums
// over bs lanes go through a per-warp scratch line.  Requires p == PP, PP | F, bs | F/PP, bs <= 32.
template <int PP>
__global__ void __launch_bounds__(SH_THREADS)
k_shp(const ShDev d, const float *__restrict__ amp, const float *__restrict__ phase, float *__restrict__ slopes,
      float *__restrict__ flux, float *__restrict__ spots) {
    using pyr::cmul;
    using pyr::fma2;
    extern __shared__ float2 sm[];
    const int F = d.F, bs = d.bs, npix = d.npix, tid = threadIdx.x;
    const int warp = tid >> 5, lane = tid & 31, Q = F / PP;
    float2 *tw = sm;                // [Q][PP]   w^(b n)
    float2 *e = tw + Q * PP;        // [PP][PP]  A exp(i phi)
    float2 *T = e + PP * PP;        // [PP][F]
    float *scr = reinterpret_cast<float *>(T + PP * F) + warp * (PP * 32);   // [NW][PP][32] column sums of a job
    __shared__ float red[4][NW];
    const int sub = blockIdx.x;
    const int sx = sub % d.ns, sy = (sub / d.ns) % d.ns, b_ = sub / (d.ns * d.ns);

    for (int i = tid; i < Q * PP; i += SH_THREADS) tw[i] = __ldg(&d.w[((i / PP) * (i % PP)) % F]);
    const float a2 = load_patch(d, amp, phase, b_, sy, sx, e);
    __syncthreads();
    for (int i = tid; i < PP * Q; i += SH_THREADS) {      // rows: (y, b) -> T[y][Q a + b], a < PP
        const int y = i / Q, b = i % Q;
        float2 v[PP];
        v[0] = e[y * PP];
#pragma unroll
        for (int x = 1; x < PP; ++x) v[x] = cmul(e[y * PP + x], tw[b * PP + x]);
        pyr::dftR<PP, -1>(v);
#pragma unroll
        for (int a = 0; a < PP; ++a) T[y * F + Q * a + b] = v[a];
    }
    __syncthreads();
    const float inv = 1.0f / ((float)F * (float)F);
    float fl = 0.f, mx = 0.f, my = 0.f;
    float *px = spots ? spots + (size_t)sub * npix * npix : nullptr;
    const int ppc = 32 / bs, CW = ppc * bs;               // pixels and columns per chunk
    const int nblk = Q / bs, nchunk = (F + CW - 1) / CW;
    for (int job = warp; job < nblk * nchunk; job += NW) {
        const int blk = job / nchunk, chunk = job % nchunk;
        const int U = chunk * CW + lane, cu = U - F / 2;
        const bool on = lane < CW && U < F;
        const int u = on ? (cu < 0 ? cu + F : cu) : 0;
        // (lanes beyond the chunk hold zeros: no selects in the loop)
        float2 t[PP], pacc[PP], srw = make_float2(0.f, 0.f);
#pragma unroll
        for (int y = 0; y < PP; ++y) {
            t[y] = on ? T[y * F + u] : make_float2(0.f, 0.f);
            pacc[y] = make_float2(0.f, 0.f);
        }
        float sn = 0.f;                                    // |f|^2 of the Nyquist row (v = F/2: a = PP/2, b = 0)
        const float2 *twb = tw + blk * bs * PP;
        float dbf = 0.f;
        for (int db = 0; db < bs; ++db, twb += PP, dbf += 1.0f) {
            float2 v[PP];
            v[0] = t[0];
#pragma unroll
            for (int y = 1; y < PP; ++y) v[y] = cmul(t[y], twb[y]);
            pyr::dftR<PP, -1>(v);                          // v[a] = f[Q a + b][u], b = blk bs + db
            float2 row = make_float2(0.f, 0.f);
#pragma unroll
            for (int a = 0; a < PP; ++a) {
                pacc[a] = fma2(v[a], v[a], pacc[a]);
                row = fma2(v[a], v[a], row);
            }
            srw = fma2(pyr::bc(dbf), row, srw);
            if (blk == 0 && db == 0) sn = v[PP / 2].x * v[PP / 2].x + v[PP / 2].y * v[PP / 2].y;
        }
        float tot = 0.f, ym = srw.x + srw.y;
#pragma unroll
        for (int a = 0; a < PP; ++a) {
            const float s = pacc[a].x + pacc[a].y;
            tot += s;
            ym = fmaf((float)(Q * ((a + PP / 2) % PP) + blk * bs - F / 2), s, ym);   // centred row of output a at db = 0
            if (px) scr[((a + PP / 2) % PP) * 32 + lane] = s;
        }
        fl += tot;
        if (cu != -F / 2) mx = fmaf((float)cu, tot, mx);  // Nyquist column: no first moment
        my += ym + (float)(F / 2) * sn;                    // Nyquist row: take it back
        if (px) {
            __syncwarp();
            for (int o = lane; o < PP * ppc; o += 32) {
                const int ap = o / ppc, seg = o % ppc, X = chunk * ppc + seg;
                if (X < npix) {
                    float a = 0.f;
                    for (int i = 0; i < bs; ++i) a += scr[ap * 32 + seg * bs + i];
                    px[((Q * ap) / bs + blk) * npix + X] = a * inv;
                }
            }
            __syncwarp();
        }
    }
    finish(d, fl, mx, my, a2, inv, sub, slopes, flux, red);
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
    float2 *d_w;
    int device;
};

extern "C" {

int sh_last_error(void) { return g_err; }
const char *sh_last_error_string(void) { return g_msg; }

sh_plan *sh_plan_create(int P, int ns, int F, int bs, int B) {
    if (P < 1 || ns < 1 || P % ns != 0) { set_err(1, "n_sub=%d must divide N_pup=%d", ns, P); return nullptr; }
    const int p = P / ns;
    if (p > 32) { set_err(2, "sub-aperture of %d pixels: at most 32 supported", p); return nullptr; }
    if (F < 4 || F > 512 || (F & 1) || F < p) { set_err(1, "F=%d must be even and in [max(p, 4), 512]", F); return nullptr; }
    if (bs < 1 || F % bs != 0) { set_err(1, "spot_binning=%d must divide F", bs); return nullptr; }
    if (B < 1 || (long long)B * ns * ns > 2147483647LL) { set_err(1, "batch=%d must be >= 1 (and B n_sub^2 < 2^31)", B); return nullptr; }
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { set_err(4, "no CUDA device: %s", cudaGetErrorString(cudaGetLastError())); return nullptr; }
    sh_plan *pl = new (std::nothrow) sh_plan();
    if (!pl) { set_err(3, "host allocation failed"); return nullptr; }
    pl->device = dev;
    pl->d_w = nullptr;
    pl->d = ShDev{P, ns, p, F, bs, F / bs, B, nullptr};
    const bool pruned = (p == 4 || p == 8 || p == 16) && F % p == 0 && (F / p) % bs == 0 && bs <= 32;
    if (pruned) {
        pl->kernel = p == 4 ? k_shp<4> : p == 8 ? k_shp<8> : k_shp<16>;
        pl->smem = (size_t)(F + p * p + p * F) * sizeof(float2) + (size_t)NW * p * 32 * sizeof(float);
    } else {
        if (F >= 128 && bs % 4 == 0) pl->kernel = k_sh<4, 4>;
        else if (F >= 64) pl->kernel = bs % 8 == 0 ? k_sh<8, 2> : bs % 4 == 0 ? k_sh<4, 2> : bs % 2 == 0 ? k_sh<2, 2> : k_sh<1, 2>;
        else pl->kernel = bs % 4 == 0 ? k_sh<4, 1> : bs % 2 == 0 ? k_sh<2, 1> : k_sh<1, 1>;
        pl->smem = (size_t)(F + p * p + p * F) * sizeof(float2) + (size_t)NW * F * sizeof(float);
    }
    if (pl->smem > 227 * 1024) { set_err(2, "p=%d, F=%d need %zu bytes of shared memory", p, F, pl->smem); delete pl; return nullptr; }
    // w[j] = exp(-2 pi i j / F), each entry from a direct sin/cos in double, rounded once
    std::vector<float2> w((size_t)F);
    for (int j = 0; j < F; ++j) {
        const double a = -2.0 * 3.14159265358979323846 * (double)j / (double)F;
        w[j] = make_float2((float)std::cos(a), (float)std::sin(a));
    }
    cudaError_t e = cudaMalloc((void **)&pl->d_w, (size_t)F * sizeof(float2));
    if (e == cudaSuccess) e = cudaMemcpy(pl->d_w, w.data(), (size_t)F * sizeof(float2), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaFuncSetAttribute((const void *)pl->kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl->smem);
    if (e != cudaSuccess) {
        set_err(e == cudaErrorMemoryAllocation ? 3 : 4, "plan setup failed: %s", cudaGetErrorString(e));
        if (pl->d_w) cudaFree(pl->d_w);
        delete pl;
        return nullptr;
    }
    pl->d.w = pl->d_w;
    return pl;
}

int sh_compute(sh_plan *pl, const float *amp, const float *phase, float *out_slopes, float *out_flux,
               float *out_spots, void *stream) {
    if (!pl || !amp || !phase || !out_slopes) return set_err(1, "sh_compute: NULL plan, amp, phase or out_slopes");
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != pl->device)
        return set_err(1, "sh_compute: the plan was created on device %d, the current device is %d", pl->device, dev);
    const ShDev &d = pl->d;
    pl->kernel<<<d.B * d.ns * d.ns, SH_THREADS, pl->smem, (cudaStream_t)stream>>>(d, amp, phase, out_slopes, out_flux, out_spots);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return set_err(4, "sh_compute: launch failed: %s", cudaGetErrorString(e));
    return 0;
}

void sh_plan_destroy(sh_plan *pl) {
    if (!pl) return;
    if (pl->d_w) cudaFree(pl->d_w);
    delete pl;
}

}  // extern "C"
