// pyr.cu -- libpyr: plan, kernels and the C ABI declared in include/pyr.h.
//
// Path (BASELINE.json:north_star; paper objects ModulatedPyramid + PyrSlopec, PAPER.md:316-317,
// 327; definition SURVEY.md 8(c)): the ideal four-face mask is separable, mask[v][u] =
// g(v) g(u), so IDFT2(mask . DFT2(E)) = C_x C_y E with the 1-D operator C = IDFT . diag(g) . DFT
// (pin P11).  The tilt of modulation point k is separable too,
// tilt_k = ty_k(y) tx_k(x).  Hence, with the pupil moved to rows/columns 0..P-1 (a cyclic
// translation of the output by o = (N-P)/2, undone when storing):
//
//   k_cols_h : for every distinct y-tilt j, every pupil column x:  R_j[:, x] = C (A e^{i phi} ty_j)[:, x]
//              (field build fused into the load; P lines per (source, j))
//   k_rows_h : for every row y', every k:  O_k[y', :] = C ( R_j(k)[y', 0:P] tx_k ),
//              I[y', :] += |O_k|^2 in registers over all k, then x-binning
//   k_rebin  : y-binning -> D, per-row valid-pixel sums (+ the slopes on small detectors, by its last CTA)
//   k_slope  : global mean + slopes (larger detectors)
//
// For the built-in mask C is evaluated in its half-band form: one forward and one inverse
// transform of length N/2 per line (pyr_kernels.cuh).  At N_fft = 2048 the same passes are
// k_field + k_cols_t + k_rows_t (row-contiguous R, bulk-copy staging, TMA stores).  k_cols / k_rows are the
// full-length, table-mask versions (custom separable masks, N = 16, N_fft not a power of two), k_g_* the three-pass
// path for general 2-D masks.  This file holds the plan, the small reduction kernels and the C ABI; the line kernels
// are instantiated per FFT size in pyr_inst.cu.  All kernels of a call are chained by programmatic dependent launch.
//
// No cuFFT, no atomics on data, no allocation or synchronisation inside pyr_compute.
#include <cuda.h>
#include <cuda_runtime.h>

#include <cmath>
#include <complex>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <algorithm>
#include <mutex>
#include <new>
#include <vector>

#include "../../include/pyr.h"
#include "pyr_kernels.cuh"

namespace pyr {

// pixels [i0, i1) (row-major over N_q x N_q) of the slope maps of source s; T-bar from the row sums in index order
// (every CTA alike)
__device__ __forceinline__ void slopes_of_source(const DevPlan &pd, int s, int i0, int i1, const float *__restrict__ D,
                                                 float *__restrict__ slopes, float *red) {
    const int Nd = pd.Nd, Nq = pd.Nq;
    const float *__restrict__ Ds = D + (size_t)s * Nd * Nd;
    // the quadrant values of up to U pixels per thread are fetched BEFORE the reduction that gives T-bar (they do not
    // depend on it): one memory round trip for the row sums and the pixels together instead of three in a row
    constexpr int U = 4;
    float Q[U][4];
    bool ok[U];
    auto fetch = [&](int base) {
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int i = base + u * 256 + (int)threadIdx.x, ii = min(i, i1 - 1);
            const int Y = ii / Nq, X = ii - Y * Nq;
            ok[u] = i < i1 && pd.valid[ii] != 0;
            Q[u][0] = __ldcg(&Ds[(size_t)Y * Nd + X]);
            Q[u][1] = __ldcg(&Ds[(size_t)Y * Nd + X + Nq]);
            Q[u][2] = __ldcg(&Ds[(size_t)(Y + Nq) * Nd + X]);
            Q[u][3] = __ldcg(&Ds[(size_t)(Y + Nq) * Nd + X + Nq]);
        }
    };
    float part = 0.f;
    for (int i = threadIdx.x; i < Nd; i += 256) part += __ldcg(&pd.partial[s * Nd + i]);
    fetch(i0);
    red[threadIdx.x] = part;
    __syncthreads();
    for (int w = 128; w > 0; w >>= 1) {
        if (threadIdx.x < w) red[threadIdx.x] += red[threadIdx.x + w];
        __syncthreads();
    }
    const float tot = red[0];
    const float Tbar = pd.n_valid > 0 ? tot / (float)pd.n_valid : 0.f;
    const float inv = Tbar > 0.f ? 1.0f / Tbar : 0.f;
    float *__restrict__ sx = slopes + (size_t)s * 2 * Nq * Nq;
    float *__restrict__ sy = sx + (size_t)Nq * Nq;
    for (int base = i0; base < i1; base += 256 * U) {
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int i = base + u * 256 + (int)threadIdx.x;
            if (i < i1) {
                const float Qa = Q[u][0], Qb = Q[u][1], Qc = Q[u][2], Qd = Q[u][3];
                sx[i] = ok[u] ? ((Qb + Qd) - (Qa + Qc)) * inv : 0.f;
                sy[i] = ok[u] ? ((Qc + Qd) - (Qa + Qb)) * inv : 0.f;
            }
        }
        if (base + 256 * U < i1) fetch(base + 256 * U);
    }
}

// ---------------------------------------------------------------- k_rebin: y-binning (+ sum of the k-chunks) + valid partial sums + slopes
// One CTA per detector row.  Small detectors (done != NULL; N_q <= 32): the CTA that finishes LAST for its source (a
// counter per source, atomicInc wrapping back to 0 -- an atomic on control flow only, never on data) also computes
// T-bar from the row sums in index order and the slopes of the whole source (a9): one launch instead of two for the
// launch-bound configurations.  D and the row sums of the other CTAs are read through L2 (__ldcg) after the fence.
// Larger detectors: k_slope (one CTA per slope row) follows as a programmatic dependent launch.
__global__ void __launch_bounds__(256) k_rebin(const DevPlan pd, float *__restrict__ D, float *__restrict__ slopes,
                                               unsigned *__restrict__ done) {
    __shared__ float red[256];
    __shared__ bool last;
    const int Yd = blockIdx.x, s = blockIdx.y;
    const int Nd = pd.Nd, Nq = pd.Nq, b = pd.b, N = pd.N;
    pdl_wait();                                    // S is complete
    float part = 0.f;
    const int T = pd.SC * b;                       // terms per detector pixel: (chunk kc, row j of the bin), kc slowest
    const size_t cstride = (size_t)pd.B * N * Nd;  // from chunk to chunk
    for (int X = threadIdx.x; X < Nd; X += 256) {
        const float *__restrict__ S = pd.S + ((size_t)s * N + (size_t)Yd * b) * Nd + X;
        const bool ok = pd.valid[(Yd % Nq) * Nq + (X % Nq)] != 0;
        float sum = 0.f;
        // eight independent loads in flight, then their sum in index order (the plain loop ran one L2 round trip per term)
        size_t off = 0;                            // of term (kc, j): kc * cstride + j * Nd, stepped without a division
        int j = 0;
        for (int t0 = 0; t0 < T; t0 += 8) {
            float v[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                v[i] = t0 + i < T ? S[off] : 0.f;
                off += Nd;
                if (++j == b) { j = 0; off += cstride - (size_t)b * Nd; }
            }
#pragma unroll
            for (int i = 0; i < 8; ++i) sum += v[i];
        }
        D[((size_t)s * Nd + Yd) * Nd + X] = sum;
        if (ok) part += sum;
    }
    // row sum over valid pixels: shuffle tree per warp, the eight warp sums in index order
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) part += __shfl_down_sync(0xffffffffu, part, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = part;
    __syncthreads();
    pdl_trigger();
    if (threadIdx.x == 0) {
        float r = 0.f;
        for (int w = 0; w < 8; ++w) r += red[w];
        pd.partial[s * Nd + Yd] = r;
    }
    if (!slopes || !done) return;
    __threadfence();                               // this CTA's D row and row sum before its tick of the counter
    __syncthreads();
    if (threadIdx.x == 0) last = atomicInc(&done[s], (unsigned)Nd - 1u) == (unsigned)Nd - 1u;
    __syncthreads();
    if (!last) return;
    __threadfence();
    slopes_of_source(pd, s, 0, Nq * Nq, D, slopes, red);
}

// ---------------------------------------------------------------- k_partial: valid-pixel row sums of a detector frame
// (PyrSlopec on detector pixels, pyr_slopes_from_pixels: the frame plays the role of D, k_slope does the rest)
__global__ void __launch_bounds__(256) k_partial(const DevPlan pd, const float *__restrict__ D) {
    __shared__ float red[256];
    const int Yd = blockIdx.x, s = blockIdx.y;
    const int Nd = pd.Nd, Nq = pd.Nq;
    pdl_trigger();
    pdl_wait();                                    // the frame is complete
    float part = 0.f;
    for (int X = threadIdx.x; X < Nd; X += 256)
        if (pd.valid[(Yd % Nq) * Nq + (X % Nq)]) part += D[((size_t)s * Nd + Yd) * Nd + X];
    red[threadIdx.x] = part;
    __syncthreads();
    for (int w = 128; w > 0; w >>= 1) {
        if (threadIdx.x < w) red[threadIdx.x] += red[threadIdx.x + w];
        __syncthreads();
    }
    if (threadIdx.x == 0) pd.partial[s * Nd + Yd] = red[0];
}

// ---------------------------------------------------------------- k_field (N_fft = 2048)
// E0[s][g][x][y] = A exp(i gscale[g] phi), column-contiguous: a1, the field build, evaluated once per pixel; the column
// kernel stages whole columns of it with bulk copies.
__global__ void __launch_bounds__(256) k_field(const DevPlan pd, const float *__restrict__ amp, const float *__restrict__ phase) {
    __shared__ float2 tile[32][33];
    const int P = pd.P, sg = blockIdx.z, s = sg / pd.NG, x0 = blockIdx.x * 32, y0 = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const float scale = pd.gscale ? __ldg(&pd.gscale[sg % pd.NG]) : 1.0f;
    float2 ap[4];                                  // all loads first: the compiler does not move them across sincosf
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int y = min(y0 + ty + 8 * i, P - 1), x = min(x0 + tx, P - 1);
        const size_t ix = ((size_t)s * P + y) * P + x;
        ap[i] = make_float2(__ldg(&amp[ix]), __ldg(&phase[ix]));
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int y = y0 + ty + 8 * i, x = x0 + tx;
        float2 e = make_float2(0.f, 0.f);
        if (y < P && x < P) {
            float sn, cs;
            sincosf(scale * ap[i].y, &sn, &cs);
            e = make_float2(ap[i].x * cs, ap[i].x * sn);
        }
        tile[ty + 8 * i][tx] = e;
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int x = x0 + ty + 8 * i, y = y0 + tx;
        if (y < P && x < P) pd.E0[((size_t)sg * P + x) * P + y] = tile[tx][ty + 8 * i];
    }
}

// ---------------------------------------------------------------- k_field_r (general masks at transform length 2048)
// E0r[s][g][y][x] = A exp(i gscale[g] phi), row-contiguous: the field build once per pixel and wavelength
__global__ void __launch_bounds__(256) k_field_r(const DevPlan pd, const float *__restrict__ amp, const float *__restrict__ phase) {
    const int P = pd.P, sg = blockIdx.y, s = sg / pd.NG;
    const float scale = pd.gscale ? __ldg(&pd.gscale[sg % pd.NG]) : 1.0f;
    for (int i = blockIdx.x * 256 + threadIdx.x; i < P * P; i += gridDim.x * 256) {
        const float a = __ldg(&amp[(size_t)s * P * P + i]);
        float sn, cs;
        sincosf(scale * __ldg(&phase[(size_t)s * P * P + i]), &sn, &cs);
        pd.E0r[(size_t)sg * P * P + i] = make_float2(a * cs, a * sn);
    }
}

// ---------------------------------------------------------------- k_slope: one CTA per slope row (after k_rebin or k_partial)
__global__ void __launch_bounds__(256) k_slope(const DevPlan pd, const float *__restrict__ D, float *__restrict__ slopes) {
    __shared__ float red[256];
    pdl_wait();                                    // D and the row sums are complete
    slopes_of_source(pd, blockIdx.y, blockIdx.x * pd.Nq, (blockIdx.x + 1) * pd.Nq, D, slopes, red);
}

// ---------------------------------------------------------------- k_fma_peak (measurement hook)
// FP32 FMA-chain microbenchmark: 8 independent packed fma.rn.f32x2 chains per thread -- the
// instruction the line kernels are made of -- CHAINS x ITERS x 4 flops per thread.  Measures what the FP32 pipes
// deliver at the clock the device actually runs; bench.py prints it next to the derived 148 x 128 x 2 x f figure.
__global__ void __launch_bounds__(256) k_fma_peak(int iters, float2 seed, float2 *__restrict__ out) {
    float2 a[8];
#pragma unroll
    for (int c = 0; c < 8; ++c) a[c] = make_float2(seed.x + 0.001f * (float)(c + threadIdx.x), seed.y - 0.001f * (float)c);
    const float2 m = make_float2(0.999f, 1.001f), b = make_float2(1e-3f, -1e-3f);
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int c = 0; c < 8; ++c) a[c] = fma2(a[c], m, b);
    }
    float2 r = a[0];
#pragma unroll
    for (int c = 1; c < 8; ++c) r = cadd(r, a[c]);
    if (r.x == 123.456f) out[blockIdx.x * blockDim.x + threadIdx.x] = r;     // never true: keeps the chains alive
}

}  // namespace pyr

// ---------------------------------------------------------------- static scratch of pyr_slopes_from_pixels_static
// The row sums that k_partial writes and k_slope reads ([B][N_det] floats) for callers that may not allocate: a
// file-scope device array of PYR_STATIC_SCRATCH_FLOATS floats (256 KB), held by every GPU that loads libpyr.so
// until the process exits.  In host code this name is a host-side stand-in, NOT a device address: the host takes
// the address with cudaGetSymbolAddress (static_scratch_ptr, below), once per device.
#define PYR_STATIC_SCRATCH_FLOATS 65536
static __device__ __align__(256) float g_static_scratch[PYR_STATIC_SCRATCH_FLOATS];

// ==================================================================== host side

#define PYR_MAX_KERNELS 8
static const char *const k_names[] = {"k_cols", "k_rows", "k_rebin", "k_slope"};

static thread_local int g_err = PYR_OK;
static thread_local char g_msg[512] = "";

static int set_err(int code, const char *fmt, ...) {
    g_err = code;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_msg, sizeof(g_msg), fmt, ap);
    va_end(ap);
    return code;
}

struct pyr_plan {
    DevPlan d;
    float r;
    int device;
    std::vector<void *> allocs;     // every device allocation, freed at destroy
    float2 *d_gx, *d_gy;            // mutable aliases of d.gx / d.gy
    unsigned char *d_valid;
    float *d_D;                     // internal D when out_intensity == NULL
    unsigned *d_done;               // [B] per-source counters of k_rebin's last-CTA slope stage (self-resetting)
    float *st_amp, *st_phase, *st_I, *st_s;   // staging for pyr_compute_host
    // double-buffered variant (pyr_compute_host_async / pyr_host_wait): two staging sets, three internal streams
    float *sa_amp[2], *sa_phase[2], *sa_I[2], *sa_s[2];
    cudaStream_t as_h2d, as_comp, as_d2h;
    cudaEvent_t aev_h2d[2], aev_comp[2], aev_d2h[2];
    bool async_ready, aslot_used[2];
    KernelSet ks_table;             // full-length kernels, table-driven mask
    int NT;                         // transform length of the table-mask kernels (= N_fft when that is a power of two)
    bool custom_mask;
    bool general_mask;              // a full N x N mask is set (pyr_plan_set_mask): three-pass path
    float2 *d_MT;                   // its device copy in position order (allocated on first use)
    float *d_Sg;                    // S of the general path: one chunk per group of kch points
    int g_chunks;
    HalfSet hs;                     // half-band-split kernels
    int cols_grid;                  // CTAs of the persistent column kernel (N_fft = 2048)
    Gen2Set g2;                     // general 2-D mask at transform length 2048: the two-halves kernels
    bool use_t2;                    // separable table masks at transform length 2048: k_field + k_h2_cols<SEP> + k_t2_rows
    float2 *d_gx2, *d_gy2;
    CUtensorMap tmR2;               // R as [B J][N][2 P floats]
    size_t t2_cols_smem, t2_rows_smem;
    void (*t2_cols)(const DevPlan, const CUtensorMap, int);
    void (*t2_rows)(const DevPlan);
    int t2_slots;                   // resident CTAs of the persistent k_t2_rows
    bool use_g2;
    int g2_grid;                    // CTAs of the persistent passes A and B (two per SM)
    pyr::Gen2Maps g2maps;
    CUtensorMap tmR, tmRring;       // R as a 3-D tensor [B J][N/2 + P][2 P floats] for k_cols_t's TMA stores (J = all / the ring)
    bool use_half;                  // built for this N (>= 32); used whenever the built-in mask is active
    std::vector<double> aye;        // effective a_y (lambda/D) of every distinct y-tilt: pyr_plan_set_double_roof rebuilds ty / hy
    bool poly;                      // more than one field group (polychromatic plan)
    int sched_jc;                   // > 0: L2-resident schedule, y-tilts per chunk (pyr_plan_set_schedule)
    int sched_chunks;
    float *d_Sc;                    // S with one slot per chunk of that schedule
    std::vector<int> jtask0;        // [J + 1] first task of every y-tilt in the sorted task list
    bool profiling;                 // record an event around every kernel (bench.py only)
    bool prof_valid;
    int prof_nk;                    // kernels launched by the last profiled call
    cudaEvent_t ev[PYR_MAX_KERNELS + 1];
};

namespace {

template <typename T>
bool dev_alloc(pyr_plan *p, T **ptr, size_t count) {
    void *q = nullptr;
    if (cudaMalloc(&q, count * sizeof(T) > 0 ? count * sizeof(T) : 16) != cudaSuccess) return false;
    p->allocs.push_back(q);
    *ptr = static_cast<T *>(q);
    return true;
}

template <typename T>
bool upload(pyr_plan *p, const T **dst, const std::vector<T> &h) {
    T *q = nullptr;
    if (!dev_alloc(p, &q, h.size())) return false;
    if (cudaMemcpy(q, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice) != cudaSuccess) return false;
    *dst = q;
    return true;
}

bool is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }

void factors(int N, int *N1, int *N2, int *N3) {
    switch (N) {
        case 16:   *N1 = 16; *N2 = 1;  *N3 = 1; break;
        case 32:   *N1 = 8;  *N2 = 4;  *N3 = 1; break;
        case 64:   *N1 = 8;  *N2 = 8;  *N3 = 1; break;
        case 128:  *N1 = 16; *N2 = 8;  *N3 = 1; break;
        case 256:  *N1 = 16; *N2 = 16; *N3 = 1; break;
        case 512:  *N1 = 4;  *N2 = 16; *N3 = 8; break;
        case 1024: *N1 = 8;  *N2 = 8;  *N3 = 16; break;
        default:   *N1 = 16; *N2 = 16; *N3 = 8; break;   // 2048
    }
}

// Where LineConv's table-mask multiply reads the value of digit-reversed position p: thread t,
// butterfly i, register q with p = (t + TPL*i)*RL + q  ->  (i*RL + q)*TPL + t (coalesced per warp).
int mask_slot(int N, int p) {
    int N1, N2, N3;
    factors(N, &N1, &N2, &N3);
    const int TPL = N / 16, RL = N3 > 1 ? N3 : (N2 > 1 ? N2 : N1);
    const int cc = p / RL, q = p % RL, t = cc % TPL, i = cc / TPL;
    return (i * RL + q) * TPL + t;
}

// 1-D mask in the table order of LineConv: position p = (k1*N2 + k2)*N3 + k3 holds frequency
// k1 + N1*k2 + N1*N2*k3 and is stored at mask_slot(p).
std::vector<float2> permute_mask(int N, const std::vector<float2> &g) {
    int N1, N2, N3;
    factors(N, &N1, &N2, &N3);
    std::vector<float2> out(N);
    for (int k1 = 0; k1 < N1; ++k1)
        for (int k2 = 0; k2 < N2; ++k2)
            for (int k3 = 0; k3 < N3; ++k3)
                out[mask_slot(N, (k1 * N2 + k2) * N3 + k3)] = g[k1 + N1 * k2 + N1 * N2 * k3];
    return out;
}

// g(u) = (-i)^|f(u)|, exact
std::vector<float2> pyramid_mask_1d(int N) {
    static const float re[4] = {1.f, 0.f, -1.f, 0.f}, im[4] = {0.f, -1.f, 0.f, 1.f};
    std::vector<float2> g(N);
    for (int u = 0; u < N; ++u) {
        int e = (u < N / 2 ? u : N - u) & 3;
        g[u] = make_float2(re[e], im[e]);
    }
    return g;
}

cudaError_t prepare_general(const KernelSet &k) {
    const void *fns[3] = {(const void *)k.gfwd, (const void *)k.gcols, (const void *)k.ginv};
    for (const void *f : fns) {
        cudaError_t e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)k.rows_smem);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

const void *cols_fn(const KernelSet &k) { return (const void *)k.cols; }
const void *cols_fn(const HalfSet &k) { return k.rowmajor ? (const void *)k.cols_t : (const void *)k.cols; }

// R[planes][rows][P] complex64 as a 3-D float32 tensor for TMA stores of (4 columns x 256 rows) boxes, 32-byte swizzle
bool make_r_map(CUtensorMap *tm, float2 *R, int planes, int rows, int P) {
    typedef CUresult (*encode_t)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                 const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                 CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static encode_t enc = nullptr;
    if (!enc) {
        cudaDriverEntryPointQueryResult qr;
        void *fn = nullptr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr) != cudaSuccess || !fn) return false;
        enc = (encode_t)fn;
    }
    const cuuint64_t dims[3] = {(cuuint64_t)2 * P, (cuuint64_t)rows, (cuuint64_t)planes};
    const cuuint64_t strides[2] = {(cuuint64_t)P * 8, (cuuint64_t)rows * P * 8};
    const cuuint32_t box[3] = {8, (cuuint32_t)pyr::TMA_BOX_ROWS, 1}, es[3] = {1, 1, 1};
    return enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, R, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_32B, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <typename SET>
cudaError_t prepare_set(const SET &k) {
    cudaError_t e = cudaFuncSetAttribute(cols_fn(k), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)k.cols_smem);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute((const void *)k.rows, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)k.rows_smem);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute((const void *)k.test, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)k.test_smem);
}

// One kernel launch; pdl: with the programmatic-stream-serialization attribute, i.e. the kernel may start while its
// predecessor in the stream drains and synchronises with it by pdl_wait() (pyr_kernels.cuh).
template <typename... KArgs, typename... Args>
cudaError_t launch(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, bool pdl, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, args...);
}

cudaError_t launch_all(pyr_plan *p, const float *amp, const float *phase, float *D, float *slopes,
                       cudaStream_t st) {
    DevPlan d = p->d;
    int nk = 0;
    // (a profiled call records an event between the kernels, which serialises them: no overlap is measured into them)
    const bool pdl = !p->profiling;
    auto mark = [&]() { if (p->profiling) cudaEventRecord(p->ev[nk], st); ++nk; };
    mark();
    if (p->general_mask) {
        // general 2-D mask: three passes per chunk of kch modulation points
        const KernelSet &k = p->ks_table;
        d.S = p->d_Sg;
        d.SC = p->g_chunks;
        if (p->use_g2) launch(pyr::k_field_r, dim3((d.P * d.P + 255) / 256, d.B * d.NG), dim3(256), 0, st, false, d, amp, phase);
        for (int c = 0; c < p->g_chunks && p->use_g2; ++c) {
            const int i0 = c * d.kch, cnt = d.M - i0 < d.kch ? d.M - i0 : d.kch, slots = d.B * cnt;
            const Gen2Set &g2 = p->g2;
            launch(g2.fwd, dim3(std::min(p->g2_grid, slots * ((d.P + 3) / 4))), dim3(128), g2.fwd_smem, st, true, d, p->g2maps.f1, i0, cnt);
            launch(g2.cols, dim3(std::min(p->g2_grid, slots * 512)), dim3(128), g2.cols_smem_base + (size_t)4 * d.P * sizeof(float2), st, true, d, p->g2maps.g, cnt);
            launch(g2.inv, dim3((d.B * d.N + 3) / 4), dim3(128), g2.inv_smem, st, true, d, cnt, c);
        }
        for (int c = 0; c < p->g_chunks && !p->use_g2; ++c) {
            const int i0 = c * d.kch, cnt = d.M - i0 < d.kch ? d.M - i0 : d.kch;
            k.gfwd<<<(d.B * cnt * d.P + k.rows_G - 1) / k.rows_G, k.rows_threads, k.rows_smem, st>>>(d, amp, phase, i0, cnt);
            k.gcols<<<(d.B * cnt * p->NT + k.rows_G - 1) / k.rows_G, k.rows_threads, k.rows_smem, st>>>(d, cnt);
            k.ginv<<<(d.B * d.N + k.rows_G - 1) / k.rows_G, k.rows_threads, k.rows_smem, st>>>(d, cnt, c);
        }
        const bool fused = d.Nq <= 32;
        launch(pyr::k_rebin, dim3(d.Nd, d.B), dim3(256), 0, st, false, d, D, slopes, fused ? p->d_done : (unsigned *)nullptr);
        if (slopes && !fused) launch(pyr::k_slope, dim3(d.Nq, d.B), dim3(256), 0, st, pdl, d, (const float *)D, slopes);
        p->prof_valid = false;
        return cudaGetLastError();
    }
    if (p->use_half && !p->custom_mask) {
        const HalfSet &h = p->hs;
        d.SC = d.TC;
        if (h.rowmajor && p->sched_jc > 0) {
            // L2-resident schedule: per chunk of sched_jc y-tilts the column pass fills one half of a two-chunk ring of R
            // and the row pass consumes it (its accumulators go to chunk slot c of S, k_rebin sums the slots)
            launch(pyr::k_field, dim3((d.P + 31) / 32, (d.P + 31) / 32, d.B * d.NG), dim3(256), 0, st, false, d, amp, phase);
            const int rows = d.N / 2 + d.P, nxb = (d.P + h.cols_G - 1) / h.cols_G;
            const int rblocks = d.B * ((rows + h.rows_G - 1) / h.rows_G);
            d.S = p->d_Sc;
            d.jring = 2 * p->sched_jc;
            for (int c = 0; c < p->sched_chunks; ++c) {
                d.cj0 = c * p->sched_jc;
                d.cjn = std::min(p->sched_jc, d.J - d.cj0);
                d.ct0 = p->jtask0[d.cj0];
                d.ctn = p->jtask0[d.cj0 + d.cjn] - d.ct0;
                d.cslot = c;
                launch(h.cols_t, dim3(std::min(p->cols_grid, d.B * nxb * d.cjn)), dim3(h.cols_threads), h.cols_smem, st, true, d, p->tmRring);
                launch(h.rows, dim3(rblocks, 1), dim3(h.rows_threads), h.rows_smem, st, true, d);
            }
            d.SC = p->sched_chunks;
            const bool fused = d.Nq <= 32;
            launch(pyr::k_rebin, dim3(d.Nd, d.B), dim3(256), 0, st, true, d, D, slopes, fused ? p->d_done : (unsigned *)nullptr);
            if (slopes && !fused) launch(pyr::k_slope, dim3(d.Nq, d.B), dim3(256), 0, st, true, d, (const float *)D, slopes);
            p->prof_valid = false;
            return cudaGetLastError();
        }
        if (h.rowmajor) {
            launch(pyr::k_field, dim3((d.P + 31) / 32, (d.P + 31) / 32, d.B * d.NG), dim3(256), 0, st, false, d, amp, phase);
            launch(h.cols_t, dim3(p->cols_grid), dim3(h.cols_threads), h.cols_smem, st, pdl, d, p->tmR);
        } else {
            launch(h.cols, dim3((d.P + h.cols_G - 1) / h.cols_G, d.B, d.hJC), dim3(h.cols_threads), h.cols_smem, st, false, d, amp, phase);
        }
        mark();
        const int rows = d.N / 2 + d.P;        // row tasks per source
        const int rblocks = h.rowmajor ? d.B * ((rows + h.rows_G - 1) / h.rows_G) : (d.B * rows + h.rows_G - 1) / h.rows_G;
        launch(h.rows, dim3(rblocks, d.TC), dim3(h.rows_threads), h.rows_smem, st, pdl, d);
    } else if (p->use_t2) {
        d.SC = d.KC;
        d.twin = !p->custom_mask;              // built-in mask: out-of-band row pairs share one line
        launch(pyr::k_field, dim3((d.P + 31) / 32, (d.P + 31) / 32, d.B * d.NG), dim3(256), 0, st, false, d, amp, phase);
        launch(p->t2_cols, dim3(std::min(p->g2_grid, d.B * d.J * ((d.P + 3) / 4))), dim3(128), p->t2_cols_smem, st, pdl, d, p->tmR2, 0);
        mark();
        const int rrows = d.twin ? d.N / 2 + d.P : d.N;
        const long long units = (long long)((d.B * rrows + 3) / 4) * d.M;
        launch(p->t2_rows, dim3((unsigned)std::min<long long>(p->t2_slots, units)), dim3(128), p->t2_rows_smem, st, pdl, d);
    } else {
        const KernelSet &k = p->ks_table;
        d.SC = d.KC;
        launch(k.cols, dim3((d.P + k.cols_G - 1) / k.cols_G, d.B, d.JC), dim3(k.cols_threads), k.cols_smem, st, false, d, amp, phase);
        mark();
        d.twin = !p->custom_mask;              // built-in mask: out-of-band row pairs share one line
        const int rrows = d.twin ? d.N / 2 + d.P : d.N;
        launch(k.rows, dim3((d.B * rrows + k.rows_G - 1) / k.rows_G, d.KC), dim3(k.rows_threads), k.rows_smem, st, pdl, d);
    }
    mark();
    const bool fused = d.Nq <= 32;
    launch(pyr::k_rebin, dim3(d.Nd, d.B), dim3(256), 0, st, pdl, d, D, slopes, fused ? p->d_done : (unsigned *)nullptr);
    mark();
    if (slopes && !fused) { launch(pyr::k_slope, dim3(d.Nq, d.B), dim3(256), 0, st, pdl, d, (const float *)D, slopes); mark(); }
    if (p->profiling) { p->prof_nk = nk - 1; p->prof_valid = true; }
    return cudaGetLastError();
}

// Split the loop (y-tilts, or task pairs) of a line kernel over `chunks` CTAs along a second
// grid axis.  Cost model: the grid runs in ceil(ctas_x * c / (SMs * resident)) waves, each as
// long as its ceil(J / c) loop iterations plus a fixed per-CTA overhead (twiddle loads, sincos,
// epilogue) worth fixed4 quarter iterations (one iteration by default; three for k_rows_h, whose
// epilogue bins and stores a whole row -- measured on C5: 3 chunks 0.690 ms, 5 chunks 0.698 ms, 1 chunk
// 0.741 ms), and every chunk of the row kernels costs k_rebin a quarter iteration (chunk_cost4, in
// quarters); take the c that minimises the total.
void pick_chunks(const void *fn, int threads, size_t smem, int ctas_x, int J, int *chunks, int *per,
                 int chunk_cost4 = 0, int fixed4 = 4) {
    int resident = 1, sms = 148, dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&resident, fn, threads, smem) != cudaSuccess || resident < 1) {
        cudaGetLastError();
        resident = 1;
    }
    const long long slots = (long long)sms * resident;
    long long best = -1;
    int best_c = 1;
    for (int c = 1; c <= J && c <= 64; ++c) {
        const int it = (J + c - 1) / c;
        const int cc = (J + it - 1) / it;          // chunks actually launched
        const long long waves = ((long long)ctas_x * cc + slots - 1) / slots;
        const long long cost = waves * (4 * it + fixed4) + (long long)chunk_cost4 * cc;
        if (best < 0 || cost < best) { best = cost; best_c = cc; }
    }
    *per = (J + best_c - 1) / best_c;
    *chunks = (J + *per - 1) / *per;
}

// 1-D mask g[N] (natural DFT order) -> the table of the length-NT transform that LineConv
// multiplies its spectrum by.  NT == N: g itself.  NT > N (N not a power of two): the operator
// out(n) = sum_m x(m) kern(n - m), kern(d) = sum_u g(u) exp(+2 pi i u d / N) (period N), acts on
// m < P and is wanted for n < N, so only kern(d), -P < d < N, matters; placed on a ring of
// length NT >= N + P - 1 (d < 0 at NT + d) those never collide, and the table is DFT_NT of
// that ring divided by NT (cyclic convolution theorem).  Double precision, O(N^2 + NT^2).
std::vector<float2> embed_mask(int N, int NT, int P, const std::vector<float2> &g) {
    if (NT == N) return g;
    const double PI2 = 6.283185307179586476925286766559;
    std::vector<double> kr(N), ki(N);
    for (int d = 0; d < N; ++d) {
        double sr = 0.0, si = 0.0;
        for (int u = 0; u < N; ++u) {
            const double a = PI2 * (double)(((long long)u * d) % N) / N;
            const double c = std::cos(a), sn = std::sin(a);
            sr += g[u].x * c - g[u].y * sn;
            si += g[u].x * sn + g[u].y * c;
        }
        kr[d] = sr; ki[d] = si;
    }
    std::vector<double> rr(NT, 0.0), ri(NT, 0.0);
    for (int d = 0; d < N; ++d) { rr[d] = kr[d]; ri[d] = ki[d]; }
    for (int d = 1; d < P; ++d) { rr[NT - d] = kr[N - d]; ri[NT - d] = ki[N - d]; }
    std::vector<float2> out(NT);
    for (int u = 0; u < NT; ++u) {
        double sr = 0.0, si = 0.0;
        for (int j = 0; j < NT; ++j) {
            if (rr[j] == 0.0 && ri[j] == 0.0) continue;
            const double a = -PI2 * (double)(((long long)u * j) % NT) / NT;
            const double c = std::cos(a), sn = std::sin(a);
            sr += rr[j] * c - ri[j] * sn;
            si += rr[j] * sn + ri[j] * c;
        }
        out[u] = make_float2((float)(sr / NT), (float)(si / NT));
    }
    return out;
}

// Transform length 2048: what the two-halves kernels (k_h2_*, k_t2_rows) share -- the radix-2 twiddles w2k, the
// 1024-point twiddle tables (built by the half-band setup when N_fft = 2048, here otherwise), the kernel set.
bool setup_halves2048(pyr_plan *p) {
    DevPlan &d = p->d;
    if (d.w2k) return true;
    const double PI = 3.14159265358979323846;
    std::vector<float2> w2k(1024);
    for (int n = 0; n < 1024; ++n) w2k[n] = make_float2((float)std::cos(-2.0 * PI * n / 2048.0), (float)std::sin(-2.0 * PI * n / 2048.0));
    bool ok = upload(p, &d.w2k, w2k);
    if (d.N == 2048) {                     // the half-band tables are those of the 1024-point line
        d.lw1 = d.hw1; d.lw2 = d.hw2;
    } else {
        std::vector<float2> hw1(1024), hw2(32);
        for (int k1 = 0; k1 < 32; ++k1)
            for (int m = 0; m < 32; ++m) {
                const double a = -2.0 * PI * (double)((long long)m * k1 % 1024) / 1024.0;
                hw1[(size_t)k1 * 32 + m] = make_float2((float)std::cos(a), (float)std::sin(a));
            }
        for (int k2 = 0; k2 < 32; ++k2) hw2[k2] = make_float2(1.f, 0.f);     // N3 = 1: unused
        ok = ok && upload(p, &d.lw1, hw1) && upload(p, &d.lw2, hw2);
    }
    const int P = d.P;
    p->g2 = pyr_pick_gen2((P <= 256) ? 4 : (P <= 512) ? 2 : 1);
    int sms = 148;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, p->device);
    p->g2_grid = 2 * sms;
    return ok;
}

int set_mask_tables(pyr_plan *p, const std::vector<float2> &gx, const std::vector<float2> &gy) {
    const int N = p->d.N, NT = p->NT;
    std::vector<float2> px = permute_mask(NT, embed_mask(N, NT, p->d.P, gx));
    std::vector<float2> py = &gx == &gy ? px : permute_mask(NT, embed_mask(N, NT, p->d.P, gy));
    if (cudaMemcpy(p->d_gx, px.data(), NT * sizeof(float2), cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(p->d_gy, py.data(), NT * sizeof(float2), cudaMemcpyHostToDevice) != cudaSuccess)
        return set_err(PYR_ECUDA, "mask upload failed: %s", cudaGetErrorString(cudaGetLastError()));
    if (p->use_t2) {
        // the same tables in the position order of the two-halves kernels: u' = (u mod 2) 1024 + u / 2 (natural at 1024)
        const std::vector<float2> ex = embed_mask(N, NT, p->d.P, gx), ey = &gx == &gy ? ex : embed_mask(N, NT, p->d.P, gy);
        std::vector<float2> x2(NT), y2(NT);
        for (int up = 0; up < NT; ++up) {
            const int u = NT == 2048 ? 2 * (up % 1024) + up / 1024 : up;
            x2[up] = ex[u];
            y2[up] = ey[u];
        }
        if (cudaMemcpy(p->d_gx2, x2.data(), NT * sizeof(float2), cudaMemcpyHostToDevice) != cudaSuccess ||
            cudaMemcpy(p->d_gy2, y2.data(), NT * sizeof(float2), cudaMemcpyHostToDevice) != cudaSuccess)
            return set_err(PYR_ECUDA, "mask upload failed: %s", cudaGetErrorString(cudaGetLastError()));
    }
    return PYR_OK;
}

}  // namespace

extern "C" {

int pyr_last_error(void) { return g_err; }
const char *pyr_last_error_string(void) { return g_msg; }

// Common plan construction.  ax, ay: the M modulation points in lambda/D (double); wt: their
// weights (>= 0); jofk[k]: index of the distinct y-tilt of point k (points with the same a_y share
// one column-pass result), J of them, whose value is taken from the first point of the group.
static pyr_plan *create_impl(int P, int N, int M, const std::vector<double> &ax_in, const std::vector<double> &ay_in,
                             const std::vector<double> &wt, const std::vector<int> &jofk, int J, int b, int B,
                             float r_record, const std::vector<double> *psc = nullptr) {
    // psc: per-point factor on the whole pupil phase (polychromatic sensor, lambda_0 / lambda): the tilt of the point
    // scales with it (effective a = psc a), the turbulent phase is scaled in the field build of its group
    std::vector<double> ax(ax_in), ay(ay_in);
    if (psc)
        for (int k = 0; k < M; ++k) { ax[k] *= (*psc)[k]; ay[k] *= (*psc)[k]; }
    if (N < 16 || N > 2048 || (N & 3)) { set_err(PYR_EINVAL, "N_fft=%d must be a multiple of 4 in [16, 2048]", N); return nullptr; }
    if (P < 2 || (P & 1) || P > N / 2) { set_err(PYR_EINVAL, "N_pup=%d must be even and in [2, N_fft/2]", P); return nullptr; }
    if (M < 1) { set_err(PYR_EINVAL, "n_mod=%d must be >= 1", M); return nullptr; }
    if (b < 1 || (N / 4) % b != 0 || (N / 4 - P / 2) % b != 0) { set_err(PYR_EINVAL, "binning=%d must divide N_fft/4 and N_fft/4 - N_pup/2", b); return nullptr; }
    if (B < 1 || B > 65535) { set_err(PYR_EINVAL, "batch=%d must be in [1, 65535]", B); return nullptr; }
    // N_fft not a power of two (the paper's 660 = 220 x 3 and 1600 = 400 x 4): the
    // length-N circulant line operator acts on P samples, so it embeds exactly in a cyclic
    // convolution of any power-of-two length NT >= N + P - 1 (set_mask_tables builds its table)
    int NT = N;
    if (!is_pow2(N)) {
        NT = 16;
        while (NT < N + P - 1) NT *= 2;
        if (NT > 2048) { set_err(PYR_EUNSUPPORTED, "N_fft=%d with N_pup=%d needs a transform longer than 2048", N, P); return nullptr; }
    }
    if (M > 65536 || (double)B * N * J * P * 8.0 > 64e9) { set_err(PYR_EUNSUPPORTED, "workspace too large"); return nullptr; }

    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { set_err(PYR_ECUDA, "no CUDA device: %s", cudaGetErrorString(cudaGetLastError())); return nullptr; }

    pyr_plan *p = new (std::nothrow) pyr_plan();
    if (!p) { set_err(PYR_ENOMEM, "host allocation failed"); return nullptr; }
    p->r = r_record;
    p->NT = NT;
    p->device = dev;
    p->profiling = false; p->prof_valid = false; p->prof_nk = 0;
    for (auto &e : p->ev) e = nullptr;
    p->async_ready = false; p->aslot_used[0] = p->aslot_used[1] = false;
    p->as_h2d = p->as_comp = p->as_d2h = nullptr;
    for (int k = 0; k < 2; ++k) { p->aev_h2d[k] = p->aev_comp[k] = p->aev_d2h[k] = nullptr; p->sa_amp[k] = p->sa_phase[k] = p->sa_I[k] = p->sa_s[k] = nullptr; }
    DevPlan &d = p->d;
    d.P = P; d.N = N; d.M = M; d.B = B; d.b = b;
    d.Nd = N / b; d.Nq = d.Nd / 2; d.o = (N - P) / 2;
    d.J = J;

    const double PI = 3.14159265358979323846;
    std::vector<int> rep(J, -1);                 // first point of every y-tilt group
    for (int k = 0; k < M; ++k)
        if (rep[jofk[k]] < 0) rep[jofk[k]] = k;
    // field groups: the distinct phase scales, in order of first appearance over j
    std::vector<float> gscale;
    std::vector<int> jgroup(J, 0);
    for (int j = 0; j < J; ++j) {
        const float sc = psc ? (float)(*psc)[rep[j]] : 1.0f;
        int g = -1;
        for (size_t i = 0; i < gscale.size(); ++i)
            if (gscale[i] == sc) { g = (int)i; break; }
        if (g < 0) { g = (int)gscale.size(); gscale.push_back(sc); }
        jgroup[j] = g;
    }
    d.NG = (int)gscale.size();
    d.gscale = nullptr; d.jgroup = nullptr;
    // (a single wavelength other than the reference one is a scaled field too: found by a random sweep -- with one
    // group the kernels used to take the scale as 1)
    const bool scaled = d.NG > 1 || gscale[0] != 1.0f;
    p->poly = scaled;
    p->aye.resize(J);
    for (int j = 0; j < J; ++j) p->aye[j] = ay[rep[j]];
    const double cp = 0.5 * (P - 1);
    // tilt phasors: x-tilt per point (its weight rides along as sqrt(w)), y-tilt per group
    std::vector<float2> tx((size_t)M * P), ty((size_t)J * P);
    for (int k = 0; k < M; ++k) {
        const double akx = ax[k], sw = std::sqrt(wt[k]);
        for (int x = 0; x < P; ++x) {
            const double a = 2.0 * PI * akx * (x - cp) / P;
            tx[(size_t)k * P + x] = make_float2((float)(sw * std::cos(a) / N), (float)(sw * std::sin(a) / N));
        }
    }
    for (int j = 0; j < J; ++j) {
        const double aky = ay[rep[j]];
        for (int y = 0; y < P; ++y) {
            const double a = 2.0 * PI * aky * (y - cp) / P;
            ty[(size_t)j * P + y] = make_float2((float)(std::cos(a) / N), (float)(std::sin(a) / N));
        }
    }
    int N1, N2, N3;
    factors(NT, &N1, &N2, &N3);
    const int S1 = NT / N1;
    std::vector<float2> tw1((size_t)NT), tw2((size_t)N2 * N3);
    for (int k1 = 0; k1 < N1; ++k1)
        for (int m = 0; m < S1; ++m) {
            const double a = -2.0 * PI * (double)((long long)m * k1 % NT) / NT;
            tw1[(size_t)k1 * S1 + m] = make_float2((float)std::cos(a), (float)std::sin(a));
        }
    for (int k2 = 0; k2 < N2; ++k2)
        for (int n3 = 0; n3 < N3; ++n3) {
            const double a = -2.0 * PI * (double)(n3 * k2 % (N2 * N3)) / (N2 * N3);
            tw2[(size_t)k2 * N3 + n3] = make_float2((float)std::cos(a), (float)std::sin(a));
        }
    std::vector<unsigned char> valid((size_t)d.Nq * d.Nq);
    const int ns = P / b;
    int nv = 0;
    for (int Y = 0; Y < d.Nq; ++Y)
        for (int X = 0; X < d.Nq; ++X) {
            const long long dy = 2 * Y - (d.Nq - 1), dx = 2 * X - (d.Nq - 1);
            const unsigned char ok = dy * dy + dx * dx <= (long long)ns * ns;
            valid[(size_t)Y * d.Nq + X] = ok;
            nv += ok;
        }
    d.n_valid = nv;

    bool ok = true;
    ok = ok && upload(p, &d.tw1, tw1) && upload(p, &d.tw2, tw2) && upload(p, &d.tx, tx) && upload(p, &d.ty, ty);
    if (scaled) ok = ok && upload(p, &d.gscale, gscale) && upload(p, &d.jgroup, jgroup);
    {
        // tasks (j, k) sorted by y-tilt, so that consecutive tasks of a row read the same row of R
        std::vector<int2> tasks;
        p->jtask0.assign(J + 1, 0);
        for (int j = 0; j < J; ++j) {
            p->jtask0[j] = (int)tasks.size();
            for (int k = 0; k < M; ++k)
                if (jofk[k] == j) tasks.push_back(make_int2(j, k));
        }
        p->jtask0[J] = (int)tasks.size();
        ok = ok && upload(p, &d.tasks, tasks);
    }
    ok = ok && dev_alloc(p, &p->d_gx, (size_t)NT) && dev_alloc(p, &p->d_gy, (size_t)NT);
    ok = ok && dev_alloc(p, &p->d_valid, valid.size());
    // kernel variants and launch geometry (needs the device: occupancy query)
    const int prune = (P <= NT / 4) ? 4 : 2;
    switch (NT) {
        case 16:   p->ks_table = pyr_pick_set_16(prune); break;
        case 32:   p->ks_table = pyr_pick_set_32(prune); break;
        case 64:   p->ks_table = pyr_pick_set_64(prune); break;
        case 128:  p->ks_table = pyr_pick_set_128(prune); break;
        case 256:  p->ks_table = pyr_pick_set_256(prune); break;
        case 512:  p->ks_table = pyr_pick_set_512(prune); break;
        case 1024: p->ks_table = pyr_pick_set_1024(prune); break;
        default:   p->ks_table = pyr_pick_set_2048(prune); break;
    }
    p->custom_mask = false;
    p->general_mask = false; p->d_MT = nullptr; p->d_Sg = nullptr; p->g_chunks = 0;
    d.MT = nullptr; d.F1 = nullptr; d.G = nullptr; d.kch = 1; d.E0 = nullptr;
    d.jring = d.cj0 = d.cjn = d.ct0 = d.ctn = d.cslot = 0;
    d.twin = 0;
    p->sched_jc = 0; p->sched_chunks = 0; p->d_Sc = nullptr;
    p->use_g2 = false; d.w2k = nullptr; d.E0r = nullptr;
    p->use_t2 = false; p->d_gx2 = p->d_gy2 = nullptr; d.gx2 = d.gy2 = nullptr;
    cudaError_t pe = prepare_set(p->ks_table);
    if (pe == cudaSuccess) pe = prepare_general(p->ks_table);
    if (pe != cudaSuccess) {
        set_err(PYR_ECUDA, "kernel setup failed: %s", cudaGetErrorString(pe));
        pyr_plan_destroy(p);
        return nullptr;
    }
    {
        const KernelSet &k = p->ks_table;
        pick_chunks((const void *)k.cols, k.cols_threads, k.cols_smem, B * ((P + k.cols_G - 1) / k.cols_G), J, &d.JC, &d.Jc);
        // (row tasks of the built-in mask: N/2 + P per source; a custom mask set later runs N rows on the same chunking)
        pick_chunks((const void *)k.rows, k.rows_threads, k.rows_smem, (B * (N / 2 + P) + k.rows_G - 1) / k.rows_G, M, &d.KC, &d.Kc, 1);
        d.SC = d.KC;
    }
    // half-band split (built-in mask, N >= 32): tables of the half-length transform, kernels, chunking
    p->use_half = false;
    d.hJC = d.TC = 1; d.hJc = J; d.Tc = M;
    d.hw1 = d.hw2 = d.hx = d.hy = nullptr;
    d.lw1 = d.lw2 = nullptr;
    if (N >= 32 && NT == N) {
        const int H = N / 2;
        const int hprune = (P <= H / 4) ? 4 : (P <= H / 2) ? 2 : 1;
        switch (N) {
            case 32:   p->hs = pyr_pick_half_32(hprune); break;
            case 64:   p->hs = pyr_pick_half_64(hprune); break;
            case 128:  p->hs = pyr_pick_half_128(hprune); break;
            case 256:  p->hs = pyr_pick_half_256(hprune); break;
            case 512:  p->hs = pyr_pick_half_512(hprune); break;
            case 1024: p->hs = pyr_pick_half_1024(hprune); break;
            default:   p->hs = pyr_pick_half_2048(hprune); break;
        }
        p->hs.cols_smem += p->hs.cols_smem_perP * P;
        if (p->hs.rowmajor)                       // T of k_cols_t: (N/2 + P) rows rounded up to whole TMA boxes x 4 columns
            p->hs.cols_smem += (size_t)((N / 2 + P + pyr::TMA_BOX_ROWS - 1) / pyr::TMA_BOX_ROWS) * pyr::TMA_BOX_ROWS * p->hs.cols_G * sizeof(float2);
        p->hs.rows_smem += p->hs.rows_smem_perP * P;
        const int H1 = p->hs.N1, H2 = p->hs.N2, H3 = p->hs.N3;
        const int T1 = H / H1;
        std::vector<float2> hw1((size_t)H), hw2((size_t)H2 * H3), hx((size_t)M * P), hy((size_t)J * P);
        for (int k1 = 0; k1 < H1; ++k1)
            for (int m = 0; m < T1; ++m) {
                const double a = -2.0 * PI * (double)((long long)m * k1 % H) / H;
                hw1[(size_t)k1 * T1 + m] = make_float2((float)std::cos(a), (float)std::sin(a));
            }
        for (int k2 = 0; k2 < H2; ++k2)
            for (int n3 = 0; n3 < H3; ++n3) {
                const double a = -2.0 * PI * (double)(n3 * k2 % (H2 * H3)) / (H2 * H3);
                hw2[(size_t)k2 * H3 + n3] = make_float2((float)std::cos(a), (float)std::sin(a));
            }
        for (int k = 0; k < M; ++k) {
            const double akx = ax[k], sw = std::sqrt(wt[k]);
            for (int x = 0; x < P; ++x) {
                const double a = 2.0 * PI * akx * (x - cp) / P - 2.0 * PI * x / N;
                hx[(size_t)k * P + x] = make_float2((float)(0.5 * sw * std::cos(a)), (float)(0.5 * sw * std::sin(a)));
            }
        }
        for (int j = 0; j < J; ++j) {
            const double aky = ay[rep[j]];
            for (int y = 0; y < P; ++y) {
                const double a = 2.0 * PI * aky * (y - cp) / P - 2.0 * PI * y / N;
                hy[(size_t)j * P + y] = make_float2((float)(0.5 * std::cos(a)), (float)(0.5 * std::sin(a)));
            }
        }
        ok = ok && upload(p, &d.hw1, hw1) && upload(p, &d.hw2, hw2) && upload(p, &d.hx, hx) && upload(p, &d.hy, hy);
        cudaError_t he = prepare_set(p->hs);
        if (he != cudaSuccess) {
            set_err(PYR_ECUDA, "kernel setup failed: %s", cudaGetErrorString(he));
            pyr_plan_destroy(p);
            return nullptr;
        }
        const HalfSet &h = p->hs;
        p->cols_grid = 0;
        if (h.rowmajor) {
            int resident = 1, sms = 148;
            cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
            if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&resident, (const void *)h.cols_t, h.cols_threads, h.cols_smem) != cudaSuccess || resident < 1) resident = 1;
            p->cols_grid = std::min(sms * resident, B * ((P + 3) / 4) * J);
            ok = ok && dev_alloc(p, &d.E0, (size_t)B * d.NG * P * P);
        } else {
            pick_chunks((const void *)h.cols, h.cols_threads, h.cols_smem, B * ((P + h.cols_G - 1) / h.cols_G), J, &d.hJC, &d.hJc);
        }
        const int hrows = N / 2 + P;
        pick_chunks((const void *)h.rows, h.rows_threads, h.rows_smem,
                    h.rowmajor ? B * ((hrows + h.rows_G - 1) / h.rows_G) : (B * hrows + h.rows_G - 1) / h.rows_G, M, &d.TC, &d.Tc, 1, 12);
        p->use_half = true;
    }
    ok = ok && dev_alloc(p, &d.R, (size_t)B * N * J * P);
    if (ok && (NT == 2048 || NT == 1024)) {
        // separable table masks at transform length 2048 / 1024 (N_fft = 1600 / 660 embedded; custom separable masks at
        // N_fft = 2048 / 1024): k_field + k_h2_cols<SEP> + k_t2_rows (one warp per line, one or two 1024-point halves)
        // instead of the 64- / 128-thread table kernels
        ok = setup_halves2048(p) && dev_alloc(p, &p->d_gx2, (size_t)NT) && dev_alloc(p, &p->d_gy2, (size_t)NT);
        if (ok && !d.E0) ok = dev_alloc(p, &d.E0, (size_t)B * d.NG * P * P);
        const bool two = NT == 2048;
        p->t2_cols = two ? p->g2.cols_sep : p->g2.cols_sep1;
        p->t2_rows = two ? p->g2.rows_sep : p->g2.rows_sep1;
        p->t2_cols_smem = (two ? p->g2.cols_smem_base : p->g2.cols_sep1_smem_base) + (size_t)4 * P * sizeof(float2);
        p->t2_rows_smem = (two ? p->g2.rows_sep_smem_base : p->g2.rows_sep1_smem_base) + (size_t)8 * P * sizeof(float2);
        ok = ok && cudaFuncSetAttribute((const void *)p->t2_cols, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->t2_cols_smem) == cudaSuccess &&
             cudaFuncSetAttribute((const void *)p->t2_rows, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->t2_rows_smem) == cudaSuccess &&
             make_r_map(&p->tmR2, d.R, B * J, N, P);
        if (ok) {
            d.gx2 = p->d_gx2; d.gy2 = p->d_gy2;
            // k_t2_rows is persistent: one CTA per resident slot, the (row block, task) sequence cut into equal ranges;
            // a row block is then covered by at most ceil(M / units per CTA) + 1 CTAs = slots of S (d.KC)
            int occ = 2, sms = 148;
            cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, p->device);
            if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, (const void *)p->t2_rows, 128, p->t2_rows_smem) != cudaSuccess || occ < 1) {
                cudaGetLastError();
                occ = 1;
            }
            p->t2_slots = sms * occ;
            auto pieces = [&](int rows) {
                const long long U = (long long)((B * rows + 3) / 4) * M, grid = std::min<long long>(p->t2_slots, U), per = U / grid;
                return (int)std::min<long long>(M, (M + per - 1) / per + 1);
            };
            d.KC = std::max(pieces(N / 2 + P), pieces(N));       // (built-in mask: row twins; custom mask: all N rows)
            d.Kc = M;
            p->use_t2 = true;
        }
    }
    const int smax = d.KC > d.TC ? d.KC : d.TC;
    if (ok && p->use_half && p->hs.rowmajor && !make_r_map(&p->tmR, d.R, B * J, N / 2 + P, P)) {
        set_err(PYR_ECUDA, "cuTensorMapEncodeTiled failed for R");
        pyr_plan_destroy(p);
        return nullptr;
    }
    ok = ok && dev_alloc(p, &d.S, (size_t)smax * B * N * d.Nd);
    ok = ok && dev_alloc(p, &d.partial, (size_t)B * d.Nd);
    ok = ok && dev_alloc(p, &p->d_D, (size_t)B * d.Nd * d.Nd);
    ok = ok && dev_alloc(p, &p->d_done, (size_t)B) && cudaMemset(p->d_done, 0, sizeof(unsigned) * (size_t)B) == cudaSuccess;
    ok = ok && dev_alloc(p, &p->st_amp, (size_t)B * P * P) && dev_alloc(p, &p->st_phase, (size_t)B * P * P);
    ok = ok && dev_alloc(p, &p->st_I, (size_t)B * d.Nd * d.Nd) && dev_alloc(p, &p->st_s, (size_t)B * 2 * d.Nq * d.Nq);
    if (!ok) {
        cudaError_t e = cudaGetLastError();
        set_err(e == cudaErrorMemoryAllocation ? PYR_ENOMEM : PYR_ECUDA, "device setup failed: %s", cudaGetErrorString(e));
        pyr_plan_destroy(p);
        return nullptr;
    }
    d.gx = p->d_gx; d.gy = p->d_gy; d.valid = p->d_valid;
    cudaError_t e = cudaMemcpy(p->d_valid, valid.data(), valid.size(), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        set_err(PYR_ECUDA, "device setup failed: %s", cudaGetErrorString(e));
        pyr_plan_destroy(p);
        return nullptr;
    }
    std::vector<float2> g = pyramid_mask_1d(N);
    if (set_mask_tables(p, g, g) != PYR_OK) { pyr_plan_destroy(p); return nullptr; }
    return p;
}

pyr_plan *pyr_plan_create(int P, int N, int M, float r, int b, int B) {
    if (M < 1) { set_err(PYR_EINVAL, "n_mod=%d must be >= 1", M); return nullptr; }
    if (!(r >= 0.f) || !std::isfinite(r)) { set_err(PYR_EINVAL, "r_mod must be finite and >= 0"); return nullptr; }
    if (M > 65536) { set_err(PYR_EUNSUPPORTED, "n_mod too large"); return nullptr; }
    // modulation points (reading S9): theta_k = 2 pi k / M on a circle of radius r, weight 1.
    // Points k and (M/2 - k) mod M have the same sin(theta), hence the same y-tilt.
    const double PI = 3.14159265358979323846;
    std::vector<double> ax(M), ay(M), wt(M, 1.0);
    for (int k = 0; k < M; ++k) {
        const double th = 2.0 * PI * k / M;
        ax[k] = (double)r * std::cos(th);
        ay[k] = (double)r * std::sin(th);
    }
    std::vector<int> jofk(M, -1);
    int J = 0;
    for (int k = 0; k < M; ++k) {
        if (jofk[k] >= 0) continue;
        jofk[k] = J;
        const int kp = (M % 2 == 0) ? ((M / 2 - k) % M + M) % M : k;
        if (kp != k && jofk[kp] < 0) jofk[kp] = J;
        ++J;
    }
    return create_impl(P, N, M, ax, ay, wt, jofk, J, b, B, r);
}

pyr_plan *pyr_plan_create_points(int P, int N, int M, const float *ax_f, const float *ay_f, const float *w_f, int b, int B) {
    if (M < 1 || !ax_f || !ay_f) { set_err(PYR_EINVAL, "pyr_plan_create_points: n_points=%d must be >= 1 and ax, ay non-NULL", M); return nullptr; }
    if (M > 65536) { set_err(PYR_EUNSUPPORTED, "n_points too large"); return nullptr; }
    std::vector<double> ax(M), ay(M), wt(M, 1.0);
    for (int k = 0; k < M; ++k) {
        ax[k] = ax_f[k]; ay[k] = ay_f[k];
        if (w_f) wt[k] = w_f[k];
        if (!std::isfinite(ax[k]) || !std::isfinite(ay[k]) || !(wt[k] >= 0.0) || !std::isfinite(wt[k])) {
            set_err(PYR_EINVAL, "pyr_plan_create_points: point %d is not finite or has a negative weight", k);
            return nullptr;
        }
    }
    // points with exactly the same a_y share one column-pass result
    std::vector<int> jofk(M, -1);
    std::vector<double> seen;
    for (int k = 0; k < M; ++k) {
        int j = -1;
        for (size_t i = 0; i < seen.size(); ++i)
            if (seen[i] == ay[k]) { j = (int)i; break; }
        if (j < 0) { j = (int)seen.size(); seen.push_back(ay[k]); }
        jofk[k] = j;
    }
    return create_impl(P, N, M, ax, ay, wt, jofk, (int)seen.size(), b, B, 0.f);
}

pyr_plan *pyr_plan_create_poly(int P, int N, int M, float r, int n_wl, const float *ratio, const float *weight, int b, int B) {
    if (M < 1 || n_wl < 1 || !ratio) { set_err(PYR_EINVAL, "pyr_plan_create_poly: n_mod=%d, n_wavelengths=%d, ratio must be non-NULL", M, n_wl); return nullptr; }
    if (!(r >= 0.f) || !std::isfinite(r)) { set_err(PYR_EINVAL, "r_mod must be finite and >= 0"); return nullptr; }
    if ((long long)M * n_wl > 65536) { set_err(PYR_EUNSUPPORTED, "n_mod * n_wavelengths too large"); return nullptr; }
    for (int l = 0; l < n_wl; ++l) {
        if (!(ratio[l] > 0.f) || !std::isfinite(ratio[l]) || (weight && (!(weight[l] >= 0.f) || !std::isfinite(weight[l])))) {
            set_err(PYR_EINVAL, "pyr_plan_create_poly: wavelength %d needs a finite ratio > 0 and weight >= 0", l);
            return nullptr;
        }
        for (int m = 0; m < l; ++m)
            if (ratio[m] == ratio[l]) { set_err(PYR_EINVAL, "pyr_plan_create_poly: wavelengths %d and %d coincide", m, l); return nullptr; }
    }
    // reading PC1: at wavelength l every modulation point of the circle, the whole pupil phase scaled by ratio[l]
    const double PI = 3.14159265358979323846;
    const int MM = M * n_wl;
    std::vector<double> ax(MM), ay(MM), wt(MM), psc(MM);
    std::vector<int> jofk(MM, -1);
    int J = 0;
    for (int l = 0; l < n_wl; ++l) {
        for (int k = 0; k < M; ++k) {
            const double th = 2.0 * PI * k / M;
            ax[l * M + k] = (double)r * std::cos(th);
            ay[l * M + k] = (double)r * std::sin(th);
            wt[l * M + k] = weight ? weight[l] : 1.0;
            psc[l * M + k] = ratio[l];
        }
        for (int k = 0; k < M; ++k) {            // k and M/2 - k share sin(theta): one y-tilt per wavelength
            if (jofk[l * M + k] >= 0) continue;
            jofk[l * M + k] = J;
            const int kp = (M % 2 == 0) ? ((M / 2 - k) % M + M) % M : k;
            if (kp != k && jofk[l * M + kp] < 0) jofk[l * M + kp] = J;
            ++J;
        }
    }
    return create_impl(P, N, MM, ax, ay, wt, jofk, J, b, B, r, &psc);
}

int pyr_plan_set_double_roof(pyr_plan *p, int enable, float kappa) {
    if (!p) return set_err(PYR_EINVAL, "pyr_plan_set_double_roof: NULL plan");
    if (!std::isfinite(kappa)) return set_err(PYR_EINVAL, "pyr_plan_set_double_roof: kappa must be finite");
    if (p->poly) return set_err(PYR_EUNSUPPORTED, "pyr_plan_set_double_roof: not defined for a polychromatic plan");
    if (p->custom_mask || p->general_mask) return set_err(PYR_EINVAL, "pyr_plan_set_double_roof: the double roof replaces the mask; restore the built-in mask first");
    // Reading DR1: roof along x in focal plane 1, quadratic pupil-plane phase q of the propagation
    // to focal plane 2, roof along y.  Both roofs and q are separable, the x part of q multiplies the OUTPUT (it drops
    // out of |.|^2) and the y part the INPUT: the sensor is the four-face path with the y-tilt phasors multiplied by
    // exp(i pi kappa (y - c_p)^2).  Exact; costs nothing per call.
    const DevPlan &d = p->d;
    const int P = d.P, N = d.N, J = d.J;
    const double PI = 3.14159265358979323846, cp = 0.5 * (P - 1), kq = enable ? (double)kappa : 0.0;
    std::vector<float2> ty((size_t)J * P), hy((size_t)J * P);
    for (int j = 0; j < J; ++j)
        for (int y = 0; y < P; ++y) {
            const double a = 2.0 * PI * p->aye[j] * (y - cp) / P + PI * kq * (y - cp) * (y - cp);
            ty[(size_t)j * P + y] = make_float2((float)(std::cos(a) / N), (float)(std::sin(a) / N));
            const double ah = a - 2.0 * PI * y / N;
            hy[(size_t)j * P + y] = make_float2((float)(0.5 * std::cos(ah)), (float)(0.5 * std::sin(ah)));
        }
    cudaError_t e = cudaMemcpy(const_cast<float2 *>(d.ty), ty.data(), ty.size() * sizeof(float2), cudaMemcpyHostToDevice);
    if (e == cudaSuccess && d.hy) e = cudaMemcpy(const_cast<float2 *>(d.hy), hy.data(), hy.size() * sizeof(float2), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return set_err(PYR_ECUDA, "pyr_plan_set_double_roof: upload failed: %s", cudaGetErrorString(e));
    return PYR_OK;
}

void pyr_plan_destroy(pyr_plan *p) {
    if (!p) return;
    if (p->as_h2d) { cudaStreamSynchronize(p->as_h2d); cudaStreamDestroy(p->as_h2d); }
    if (p->as_comp) { cudaStreamSynchronize(p->as_comp); cudaStreamDestroy(p->as_comp); }
    if (p->as_d2h) { cudaStreamSynchronize(p->as_d2h); cudaStreamDestroy(p->as_d2h); }
    for (int k = 0; k < 2; ++k) {
        if (p->aev_h2d[k]) cudaEventDestroy(p->aev_h2d[k]);
        if (p->aev_comp[k]) cudaEventDestroy(p->aev_comp[k]);
        if (p->aev_d2h[k]) cudaEventDestroy(p->aev_d2h[k]);
    }
    for (void *q : p->allocs) cudaFree(q);
    for (auto &e : p->ev) if (e) cudaEventDestroy(e);
    delete p;
}

int pyr_compute(pyr_plan *p, const float *amp, const float *phase, float *out_I, float *out_s, void *stream) {
    if (!p || !amp || !phase) return set_err(PYR_EINVAL, "pyr_compute: NULL plan, amp or phase");
    if (!out_I && !out_s) return set_err(PYR_EINVAL, "pyr_compute: both outputs NULL");
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != p->device)
        return set_err(PYR_EINVAL, "pyr_compute: the plan was created on device %d, the current device is %d", p->device, dev);
    float *D = out_I ? out_I : p->d_D;
    cudaError_t e = launch_all(p, amp, phase, D, out_s, (cudaStream_t)stream);
    if (e != cudaSuccess) return set_err(PYR_ECUDA, "pyr_compute: launch failed: %s", cudaGetErrorString(e));
    return PYR_OK;
}

int pyr_slopes_from_pixels(pyr_plan *p, const float *pixels, float *out_s, void *stream) {
    if (!p || !pixels || !out_s) return set_err(PYR_EINVAL, "pyr_slopes_from_pixels: NULL argument");
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != p->device)
        return set_err(PYR_EINVAL, "pyr_slopes_from_pixels: the plan was created on device %d, the current device is %d", p->device, dev);
    const DevPlan &d = p->d;
    // (k_partial waits for the kernel that wrote the frame, k_slope for k_partial: programmatic dependent launches)
    launch(pyr::k_partial, dim3(d.Nd, d.B), dim3(256), 0, (cudaStream_t)stream, true, d, pixels);
    launch(pyr::k_slope, dim3(d.Nq, d.B), dim3(256), 0, (cudaStream_t)stream, true, d, pixels, (float *)out_s);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return set_err(PYR_ECUDA, "pyr_slopes_from_pixels: launch failed: %s", cudaGetErrorString(e));
    return PYR_OK;
}

// ---------------------------------------------------------------- the entry point that allocates nothing
// Device address of g_static_scratch on the current device, looked up once per device (with that device current)
// by cudaGetSymbolAddress and kept; no cudaMalloc / cudaFree anywhere on this path.
static int static_scratch_ptr(float **out, const char *who) {
    enum { MAX_DEV = 64 };
    static float *ptrs[MAX_DEV];                   // guarded by the mutex below
    static std::mutex mu;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MAX_DEV)
        return set_err(PYR_ECUDA, "%s: no usable current CUDA device (%s)", who, cudaGetErrorString(cudaGetLastError()));
    std::lock_guard<std::mutex> lock(mu);
    if (!ptrs[dev]) {
        float *ptr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void **)&ptr, g_static_scratch);
        if (e != cudaSuccess || !ptr)
            return set_err(PYR_ECUDA, "%s: cudaGetSymbolAddress(static scratch) failed on device %d: %s", who, dev, cudaGetErrorString(e));
        ptrs[dev] = ptr;
    }
    *out = ptrs[dev];
    return PYR_OK;
}

int pyr_static_scratch_init(void) {
    float *ptr = nullptr;
    return static_scratch_ptr(&ptr, "pyr_static_scratch_init");
}

int pyr_slopes_from_pixels_static(int N_det, int batch, const float *pixels, const unsigned char *valid, int n_valid,
                                  float *out_s, void *stream) {
    if (!pixels || !valid || !out_s) return set_err(PYR_EINVAL, "pyr_slopes_from_pixels_static: NULL argument");
    if (N_det < 2 || (N_det & 1) || batch < 1 || batch > 65535 || n_valid < 0 || (long long)n_valid > (long long)(N_det / 2) * (N_det / 2))
        return set_err(PYR_EINVAL, "pyr_slopes_from_pixels_static: N_det=%d (even, >= 2) batch=%d (1..65535) n_valid=%d", N_det, batch, n_valid);
    if ((long long)batch * N_det > PYR_STATIC_SCRATCH_FLOATS)
        return set_err(PYR_EUNSUPPORTED, "pyr_slopes_from_pixels_static: batch * N_det = %lld exceeds the static scratch of %d floats; use a plan and pyr_slopes_from_pixels",
                       (long long)batch * N_det, PYR_STATIC_SCRATCH_FLOATS);
    float *scratch = nullptr;
    const int rc = static_scratch_ptr(&scratch, "pyr_slopes_from_pixels_static");
    if (rc != PYR_OK) return rc;
    // the two kernels of pyr_slopes_from_pixels on a plan-less DevPlan: only these fields are read.  Every row sum of
    // [0, batch * N_det) is overwritten by k_partial before k_slope reads it: nothing needs clearing between calls.
    DevPlan d = {};
    d.B = batch; d.Nd = N_det; d.Nq = N_det / 2; d.n_valid = n_valid;
    d.valid = valid;
    d.partial = scratch;
    launch(pyr::k_partial, dim3(d.Nd, d.B), dim3(256), 0, (cudaStream_t)stream, true, d, pixels);
    launch(pyr::k_slope, dim3(d.Nq, d.B), dim3(256), 0, (cudaStream_t)stream, true, d, pixels, (float *)out_s);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return set_err(PYR_ECUDA, "pyr_slopes_from_pixels_static: launch failed: %s", cudaGetErrorString(e));
    return PYR_OK;
}

int pyr_compute_host(pyr_plan *p, const float *amp_h, const float *phase_h, float *out_I_h, float *out_s_h, void *stream) {
    if (!p || !amp_h || !phase_h) return set_err(PYR_EINVAL, "pyr_compute_host: NULL plan, amp or phase");
    if (!out_I_h && !out_s_h) return set_err(PYR_EINVAL, "pyr_compute_host: both outputs NULL");
    const DevPlan &d = p->d;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t nin = (size_t)d.B * d.P * d.P * sizeof(float);
    const size_t nI = (size_t)d.B * d.Nd * d.Nd * sizeof(float), ns = (size_t)d.B * 2 * d.Nq * d.Nq * sizeof(float);
    cudaError_t e = cudaMemcpyAsync(p->st_amp, amp_h, nin, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(p->st_phase, phase_h, nin, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return set_err(PYR_ECUDA, "pyr_compute_host: H2D failed: %s", cudaGetErrorString(e));
    int rc = pyr_compute(p, p->st_amp, p->st_phase, out_I_h ? p->st_I : nullptr, out_s_h ? p->st_s : nullptr, stream);
    if (rc != PYR_OK) return rc;
    if (out_I_h) e = cudaMemcpyAsync(out_I_h, p->st_I, nI, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && out_s_h) e = cudaMemcpyAsync(out_s_h, p->st_s, ns, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return set_err(PYR_ECUDA, "pyr_compute_host: D2H/sync failed: %s", cudaGetErrorString(e));
    return PYR_OK;
}

// Double-buffered end-to-end variant: slot k = 0, 1 owns a staging set; the H2D copy of a call, its kernels and its
// D2H copy run on three internal streams chained by events, so the copies of call i + 1 overlap the kernels of call i.
int pyr_compute_host_async(pyr_plan *p, const float *amp_h, const float *phase_h, float *out_I_h, float *out_s_h, int slot) {
    if (!p || !amp_h || !phase_h) return set_err(PYR_EINVAL, "pyr_compute_host_async: NULL plan, amp or phase");
    if (!out_I_h && !out_s_h) return set_err(PYR_EINVAL, "pyr_compute_host_async: both outputs NULL");
    if (slot < 0 || slot > 1) return set_err(PYR_EINVAL, "pyr_compute_host_async: slot must be 0 or 1");
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != p->device)
        return set_err(PYR_EINVAL, "pyr_compute_host_async: the plan was created on device %d, the current device is %d", p->device, dev);
    const DevPlan &d = p->d;
    const size_t nin = (size_t)d.B * d.P * d.P, nI = (size_t)d.B * d.Nd * d.Nd, ns = (size_t)d.B * 2 * d.Nq * d.Nq;
    if (!p->async_ready) {                       // first use: streams, events, the two staging sets
        bool ok = cudaStreamCreateWithFlags(&p->as_h2d, cudaStreamNonBlocking) == cudaSuccess &&
                  cudaStreamCreateWithFlags(&p->as_comp, cudaStreamNonBlocking) == cudaSuccess &&
                  cudaStreamCreateWithFlags(&p->as_d2h, cudaStreamNonBlocking) == cudaSuccess;
        for (int k = 0; k < 2 && ok; ++k) {
            ok = cudaEventCreateWithFlags(&p->aev_h2d[k], cudaEventDisableTiming) == cudaSuccess &&
                 cudaEventCreateWithFlags(&p->aev_comp[k], cudaEventDisableTiming) == cudaSuccess &&
                 cudaEventCreateWithFlags(&p->aev_d2h[k], cudaEventDisableTiming) == cudaSuccess &&
                 dev_alloc(p, &p->sa_amp[k], nin) && dev_alloc(p, &p->sa_phase[k], nin) &&
                 dev_alloc(p, &p->sa_I[k], nI) && dev_alloc(p, &p->sa_s[k], ns);
        }
        if (!ok) return set_err(PYR_ECUDA, "pyr_compute_host_async: setup failed: %s", cudaGetErrorString(cudaGetLastError()));
        p->async_ready = true;
    }
    const int k = slot;
    cudaError_t e = cudaSuccess;
    // inputs of slot k are free once the kernels of its previous call have run
    if (p->aslot_used[k]) e = cudaStreamWaitEvent(p->as_h2d, p->aev_comp[k], 0);
    if (e == cudaSuccess) e = cudaMemcpyAsync(p->sa_amp[k], amp_h, nin * sizeof(float), cudaMemcpyHostToDevice, p->as_h2d);
    if (e == cudaSuccess) e = cudaMemcpyAsync(p->sa_phase[k], phase_h, nin * sizeof(float), cudaMemcpyHostToDevice, p->as_h2d);
    if (e == cudaSuccess) e = cudaEventRecord(p->aev_h2d[k], p->as_h2d);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(p->as_comp, p->aev_h2d[k], 0);
    // outputs of slot k are free once its previous D2H copy is done
    if (e == cudaSuccess && p->aslot_used[k]) e = cudaStreamWaitEvent(p->as_comp, p->aev_d2h[k], 0);
    if (e != cudaSuccess) return set_err(PYR_ECUDA, "pyr_compute_host_async: H2D failed: %s", cudaGetErrorString(e));
    e = launch_all(p, p->sa_amp[k], p->sa_phase[k], out_I_h ? p->sa_I[k] : p->d_D, out_s_h ? p->sa_s[k] : nullptr, p->as_comp);
    if (e == cudaSuccess) e = cudaEventRecord(p->aev_comp[k], p->as_comp);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(p->as_d2h, p->aev_comp[k], 0);
    if (e == cudaSuccess && out_I_h) e = cudaMemcpyAsync(out_I_h, p->sa_I[k], nI * sizeof(float), cudaMemcpyDeviceToHost, p->as_d2h);
    if (e == cudaSuccess && out_s_h) e = cudaMemcpyAsync(out_s_h, p->sa_s[k], ns * sizeof(float), cudaMemcpyDeviceToHost, p->as_d2h);
    if (e == cudaSuccess) e = cudaEventRecord(p->aev_d2h[k], p->as_d2h);
    if (e != cudaSuccess) return set_err(PYR_ECUDA, "pyr_compute_host_async: launch failed: %s", cudaGetErrorString(e));
    p->aslot_used[k] = true;
    return PYR_OK;
}

int pyr_host_wait(pyr_plan *p, int slot) {
    if (!p || slot < 0 || slot > 1) return set_err(PYR_EINVAL, "pyr_host_wait: bad argument");
    if (!p->async_ready || !p->aslot_used[slot]) return PYR_OK;
    cudaError_t e = cudaEventSynchronize(p->aev_d2h[slot]);
    if (e != cudaSuccess) return set_err(PYR_ECUDA, "pyr_host_wait: %s", cudaGetErrorString(e));
    return PYR_OK;
}

int pyr_plan_set_schedule(pyr_plan *p, int l2_resident, int j_per_chunk) {
    if (!p) return set_err(PYR_EINVAL, "pyr_plan_set_schedule: NULL plan");
    if (!l2_resident) { p->sched_jc = 0; return PYR_OK; }
    if (!(p->use_half && p->hs.rowmajor)) return set_err(PYR_EUNSUPPORTED, "pyr_plan_set_schedule: the L2-resident schedule exists for N_fft = 2048 only");
    const DevPlan &d = p->d;
    if (j_per_chunk <= 0) {
        // two chunks of R (B x jc x (N/2 + P) x P complex64) must stay in L2 beside everything else: 80 MB
        const double per_j = (double)d.B * (d.N / 2 + d.P) * d.P * 8.0;
        j_per_chunk = (int)(80e6 / (2.0 * per_j));
        if (j_per_chunk < 1) j_per_chunk = 1;
    }
    if (j_per_chunk > d.J) j_per_chunk = d.J;
    const int chunks = (d.J + j_per_chunk - 1) / j_per_chunk;
    if (chunks > p->sched_chunks) {
        float *sc = nullptr;
        if (!dev_alloc(p, &sc, (size_t)chunks * d.B * d.N * d.Nd))
            return set_err(PYR_ENOMEM, "pyr_plan_set_schedule: %s", cudaGetErrorString(cudaGetLastError()));
        p->d_Sc = sc;
    }
    if (!make_r_map(&p->tmRring, p->d.R, d.B * 2 * j_per_chunk, d.N / 2 + d.P, d.P))
        return set_err(PYR_ECUDA, "pyr_plan_set_schedule: cuTensorMapEncodeTiled failed");
    p->sched_jc = j_per_chunk;
    p->sched_chunks = chunks;
    return PYR_OK;
}

int pyr_plan_set_valid(pyr_plan *p, const unsigned char *host_valid) {
    if (!p || !host_valid) return set_err(PYR_EINVAL, "pyr_plan_set_valid: NULL argument");
    const size_t n = (size_t)p->d.Nq * p->d.Nq;
    int nv = 0;
    std::vector<unsigned char> v(n);
    for (size_t i = 0; i < n; ++i) { v[i] = host_valid[i] ? 1 : 0; nv += v[i]; }
    if (cudaMemcpy(p->d_valid, v.data(), n, cudaMemcpyHostToDevice) != cudaSuccess)
        return set_err(PYR_ECUDA, "pyr_plan_set_valid: upload failed: %s", cudaGetErrorString(cudaGetLastError()));
    p->d.n_valid = nv;
    return PYR_OK;
}

int pyr_plan_set_mask_separable(pyr_plan *p, const float *gx_ri, const float *gy_ri) {
    if (!p) return set_err(PYR_EINVAL, "pyr_plan_set_mask_separable: NULL plan");
    const int N = p->d.N;
    if (!gx_ri && !gy_ri) {
        std::vector<float2> g = pyramid_mask_1d(N);
        p->custom_mask = false;
        return set_mask_tables(p, g, g);
    }
    if (!gx_ri || !gy_ri) return set_err(PYR_EINVAL, "pyr_plan_set_mask_separable: give both masks or neither");
    std::vector<float2> gx(N), gy(N);
    for (int u = 0; u < N; ++u) {
        gx[u] = make_float2(gx_ri[2 * u], gx_ri[2 * u + 1]);
        gy[u] = make_float2(gy_ri[2 * u], gy_ri[2 * u + 1]);
    }
    p->custom_mask = true;
    return set_mask_tables(p, gx, gy);
}

int pyr_plan_set_mask(pyr_plan *p, const float *mask_ri) {
    if (!p) return set_err(PYR_EINVAL, "pyr_plan_set_mask: NULL plan");
    if (!mask_ri) { p->general_mask = false; return PYR_OK; }
    DevPlan &d = p->d;
    const int N = d.N, NT = p->NT, P = d.P, B = d.B, M = d.M;
    if (!p->d_MT) {
        // chunk the modulation points so that G stays below ~512 MB.  Larger chunks measured faster on C5, with the
        // two-halves kernels too: 4.91 / 4.02 / 3.59 / 3.33 / 3.34 ms at 1 / 2 / 4 / 8 / 16 points per chunk -- an
        // L2-sized G (1 point: 67 MB) loses more to the short grids and the extra launches than it saves in DRAM traffic
        const double per_point = (double)B * N * NT * sizeof(float2);
        int kch = (int)(536870912.0 / per_point);
        if (kch < 1) kch = 1;
        if (kch > M) kch = M;
        const int chunks = (M + kch - 1) / kch;
        const int PT = (P + pyr::RT - 1) / pyr::RT;
        bool ok = dev_alloc(p, &p->d_MT, (size_t)NT * NT) &&
                  dev_alloc(p, &d.F1, (size_t)B * kch * PT * NT * pyr::RT) &&
                  dev_alloc(p, &d.G, (size_t)B * kch * N * NT) &&
                  dev_alloc(p, &p->d_Sg, (size_t)chunks * B * N * d.Nd);
        if (!ok) {
            cudaError_t e = cudaGetLastError();
            p->d_MT = nullptr;
            return set_err(e == cudaErrorMemoryAllocation ? PYR_ENOMEM : PYR_ECUDA,
                           "pyr_plan_set_mask: workspace allocation failed: %s", cudaGetErrorString(e));
        }
        d.MT = p->d_MT; d.kch = kch; p->g_chunks = chunks;
        if (NT == 2048) {
            // transform length 2048: the two-halves kernels (k_h2_*): their tables, tensor maps, attributes
            bool ok2 = setup_halves2048(p) && dev_alloc(p, &d.E0r, (size_t)B * d.NG * P * P);
            const size_t cols_smem = p->g2.cols_smem_base + (size_t)4 * P * sizeof(float2);
            cudaError_t ge = cudaFuncSetAttribute((const void *)p->g2.fwd, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->g2.fwd_smem);
            if (ge == cudaSuccess) ge = cudaFuncSetAttribute((const void *)p->g2.cols, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cols_smem);
            if (ge == cudaSuccess) ge = cudaFuncSetAttribute((const void *)p->g2.inv, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->g2.inv_smem);
            ok2 = ok2 && ge == cudaSuccess && make_r_map(&p->g2maps.f1, d.F1, B * kch, 2048, P) &&
                  make_r_map(&p->g2maps.g, d.G, B * kch, N, NT);
            if (!ok2) return set_err(PYR_ECUDA, "pyr_plan_set_mask: setup of the 2048-point kernels failed: %s", cudaGetErrorString(cudaGetLastError()));
            p->use_g2 = true;
        }
    }
    // The mask as the multiplier of the length-NT 2-D transform, natural frequency order.
    // NT == N: the mask itself.  NT > N (N_fft not a power of two): as embed_mask, in two dimensions --
    // kern(dy, dx) = sum_{v,u} mask[v][u] exp(+2 pi i (u dx + v dy) / N) is needed for -P < dy, dx < N,
    // goes on an NT x NT ring, and the multiplier is DFT2_NT(ring) / NT^2.  Double precision.
    typedef std::complex<double> cd;
    std::vector<cd> mfull((size_t)NT * NT);
    if (NT == N) {
        for (size_t i = 0; i < (size_t)N * N; ++i) mfull[i] = cd(mask_ri[2 * i], mask_ri[2 * i + 1]);
    } else {
        const double PI2 = 6.283185307179586476925286766559;
        // kern = N-point inverse-sign DFT of the mask along both axes, O(N^2 log N): decimation in time over the
        // prime factors of N (660 = 2^2 3 5 11, 1600 = 2^6 5^2), a prime length by the direct sum
        std::vector<cd> wN(N);
        for (int j = 0; j < N; ++j) wN[j] = cd(std::cos(PI2 * j / N), std::sin(PI2 * j / N));
        std::vector<cd> scratch(N), line(N), outl(N);
        struct Rec {
            static void run(int n, const cd *in, int is, cd *out, const std::vector<cd> &w, int N0, cd *tmp) {
                if (n == 1) { out[0] = in[0]; return; }
                int p = n;
                for (int f = 2; f * f <= n; ++f) if (n % f == 0) { p = f; break; }
                const int m = n / p, ws = N0 / n;
                if (p == n) {
                    for (int u = 0; u < n; ++u) {
                        cd acc(0.0, 0.0);
                        int e = 0;
                        for (int x = 0; x < n; ++x) { acc += in[(size_t)x * is] * w[(size_t)e * ws]; e += u; if (e >= n) e -= n; }
                        out[u] = acc;
                    }
                    return;
                }
                for (int r = 0; r < p; ++r) run(m, in + (size_t)r * is, is * p, out + (size_t)r * m, w, N0, tmp);
                for (int k = 0; k < m; ++k) {
                    for (int r = 0; r < p; ++r) tmp[r] = out[(size_t)r * m + k] * w[(size_t)((long long)r * k % n) * ws];
                    for (int q = 0; q < p; ++q) {
                        cd acc(0.0, 0.0);
                        for (int r = 0; r < p; ++r) acc += tmp[r] * w[(size_t)(r * q % p) * (N0 / p)];
                        out[(size_t)k + (size_t)q * m] = acc;
                    }
                }
            }
        };
        std::vector<cd> k2((size_t)N * N);
        for (int v = 0; v < N; ++v) {                   // along u -> dx
            for (int u = 0; u < N; ++u) line[u] = cd(mask_ri[2 * ((size_t)v * N + u)], mask_ri[2 * ((size_t)v * N + u) + 1]);
            Rec::run(N, line.data(), 1, outl.data(), wN, N, scratch.data());
            for (int dx = 0; dx < N; ++dx) k2[(size_t)v * N + dx] = outl[dx];
        }
        for (int dx = 0; dx < N; ++dx) {                // along v -> dy
            for (int v = 0; v < N; ++v) line[v] = k2[(size_t)v * N + dx];
            Rec::run(N, line.data(), 1, outl.data(), wN, N, scratch.data());
            for (int dy = 0; dy < N; ++dy) k2[(size_t)dy * N + dx] = outl[dy];
        }
        std::vector<cd> ring((size_t)NT * NT, cd(0.0, 0.0));
        for (int dy = -(P - 1); dy < N; ++dy)
            for (int dx = -(P - 1); dx < N; ++dx)
                ring[(size_t)((dy + NT) % NT) * NT + (dx + NT) % NT] = k2[(size_t)((dy + N) % N) * N + (dx + N) % N];
        // DFT2_NT by rows then columns with an iterative radix-2 FFT (NT is a power of two)
        auto fft = [&](cd *a, int stride) {
            for (int i = 1, j = 0; i < NT; ++i) {
                int bit = NT >> 1;
                for (; j & bit; bit >>= 1) j ^= bit;
                j ^= bit;
                if (i < j) std::swap(a[(size_t)i * stride], a[(size_t)j * stride]);
            }
            for (int len = 2; len <= NT; len <<= 1) {
                for (int i = 0; i < NT; i += len)
                    for (int k = 0; k < len / 2; ++k) {
                        const double ang = -PI2 * k / len;
                        const cd w(std::cos(ang), std::sin(ang));
                        const cd x = a[(size_t)(i + k) * stride], y = a[(size_t)(i + k + len / 2) * stride] * w;
                        a[(size_t)(i + k) * stride] = x + y;
                        a[(size_t)(i + k + len / 2) * stride] = x - y;
                    }
            }
        };
        for (int y = 0; y < NT; ++y) fft(&ring[(size_t)y * NT], 1);
        for (int x = 0; x < NT; ++x) fft(&ring[x], NT);
        const double sc = 1.0 / ((double)NT * NT);
        for (size_t i = 0; i < ring.size(); ++i) mfull[i] = ring[i] * sc;
    }
    // MT[p][slot(pv)] = mfull[v(pv)][u(p)]: p, pv digit-reversed positions; along v in LineConv's table order
    int N1, N2, N3;
    factors(NT, &N1, &N2, &N3);
    std::vector<int> freq(NT);
    for (int k1 = 0; k1 < N1; ++k1)
        for (int k2 = 0; k2 < N2; ++k2)
            for (int k3 = 0; k3 < N3; ++k3) freq[(k1 * N2 + k2) * N3 + k3] = k1 + N1 * k2 + N1 * N2 * k3;
    std::vector<int> slot(NT);
    for (int pv = 0; pv < NT; ++pv) slot[pv] = mask_slot(NT, pv);
    std::vector<float2> mt((size_t)NT * NT);
    if (p->use_g2) {
        // two-halves kernels: position u' = (u mod 2) 1024 + u / 2 on both axes, MT[u'][v'] = mask[v][u]
        for (int up = 0; up < NT; ++up)
            for (int vp = 0; vp < NT; ++vp) {
                const int u = 2 * (up % 1024) + up / 1024, v = 2 * (vp % 1024) + vp / 1024;
                const cd m = mfull[(size_t)v * NT + u];
                mt[(size_t)up * NT + vp] = make_float2((float)m.real(), (float)m.imag());
            }
    } else
    for (int pp = 0; pp < NT; ++pp)
        for (int pv = 0; pv < NT; ++pv) {
            const cd m = mfull[(size_t)freq[pv] * NT + freq[pp]];
            mt[(size_t)pp * NT + slot[pv]] = make_float2((float)m.real(), (float)m.imag());
        }
    if (cudaMemcpy(p->d_MT, mt.data(), mt.size() * sizeof(float2), cudaMemcpyHostToDevice) != cudaSuccess)
        return set_err(PYR_ECUDA, "pyr_plan_set_mask: upload failed: %s", cudaGetErrorString(cudaGetLastError()));
    p->general_mask = true;
    return PYR_OK;
}

int pyr_plan_get_dims(const pyr_plan *p, int *N_det, int *N_q, int *n_valid) {
    if (!p) return set_err(PYR_EINVAL, "pyr_plan_get_dims: NULL plan");
    if (N_det) *N_det = p->d.Nd;
    if (N_q) *N_q = p->d.Nq;
    if (n_valid) *n_valid = p->d.n_valid;
    return PYR_OK;
}

int pyr_test_line_conv(pyr_plan *p, const float *in_ri, float *out_ri, int nlines, void *stream) {
    if (!p || !in_ri || !out_ri || nlines < 1) return set_err(PYR_EINVAL, "pyr_test_line_conv: bad argument");
    if (p->use_half && !p->custom_mask) {
        const HalfSet &k = p->hs;
        k.test<<<(nlines + k.test_G - 1) / k.test_G, k.test_threads, k.test_smem, (cudaStream_t)stream>>>(
            p->d, (const float2 *)in_ri, (float2 *)out_ri, nlines);
    } else {
        const KernelSet &k = p->ks_table;
        k.test<<<(nlines + k.test_G - 1) / k.test_G, k.test_threads, k.test_smem, (cudaStream_t)stream>>>(
            p->d, (const float2 *)in_ri, (float2 *)out_ri, nlines);
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return set_err(PYR_ECUDA, "pyr_test_line_conv: launch failed: %s", cudaGetErrorString(e));
    return PYR_OK;
}

int pyr_plan_launches_per_compute(const pyr_plan *p) {
    if (!p) return 0;
    const int tail = p->d.Nq <= 32 ? 1 : 2;           // k_rebin (+ k_slope on larger detectors)
    if (!p->general_mask && p->use_half && !p->custom_mask && p->hs.rowmajor && p->sched_jc > 0)
        return 1 + 2 * p->sched_chunks + tail;
    if (p->general_mask) return 3 * p->g_chunks + tail + (p->use_g2 ? 1 : 0);
    if (!(p->use_half && !p->custom_mask) && p->use_t2) return 3 + tail;               // k_field + the two table passes
    return ((p->use_half && !p->custom_mask && p->hs.rowmajor) ? 3 : 2) + tail;     // + k_field at N_fft = 2048
}

int pyr_plan_set_profiling(pyr_plan *p, int enable) {
    if (!p) return set_err(PYR_EINVAL, "pyr_plan_set_profiling: NULL plan");
    if (enable && !p->ev[0]) {
        for (auto &e : p->ev)
            if (cudaEventCreate(&e) != cudaSuccess)
                return set_err(PYR_ECUDA, "pyr_plan_set_profiling: %s", cudaGetErrorString(cudaGetLastError()));
    }
    p->profiling = enable != 0;
    p->prof_valid = false;
    return PYR_OK;
}

int pyr_plan_last_kernel_ms(pyr_plan *p, float *ms, int n) {
    if (!p || !ms || n < 0) return -1;
    if (!p->prof_valid) { set_err(PYR_EINVAL, "pyr_plan_last_kernel_ms: no profiled call yet"); return -1; }
    if (cudaEventSynchronize(p->ev[p->prof_nk]) != cudaSuccess) {
        set_err(PYR_ECUDA, "pyr_plan_last_kernel_ms: %s", cudaGetErrorString(cudaGetLastError()));
        return -1;
    }
    for (int i = 0; i < p->prof_nk && i < n; ++i)
        if (cudaEventElapsedTime(&ms[i], p->ev[i], p->ev[i + 1]) != cudaSuccess) {
            set_err(PYR_ECUDA, "pyr_plan_last_kernel_ms: %s", cudaGetErrorString(cudaGetLastError()));
            return -1;
        }
    return p->prof_nk;
}

int pyr_measure_fp32_peak(float *tflops, float *sm_mhz_effective) {
    if (!tflops) return set_err(PYR_EINVAL, "pyr_measure_fp32_peak: NULL argument");
    int dev = 0, sms = 148;
    if (cudaGetDevice(&dev) != cudaSuccess) return set_err(PYR_ECUDA, "no CUDA device: %s", cudaGetErrorString(cudaGetLastError()));
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    float2 *out = nullptr;
    const int ctas = sms * 8, threads = 256, iters = 4096;
    if (cudaMalloc((void **)&out, sizeof(float2) * (size_t)ctas * threads) != cudaSuccess)
        return set_err(PYR_ENOMEM, "pyr_measure_fp32_peak: %s", cudaGetErrorString(cudaGetLastError()));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    float best = 1e30f;
    for (int rep = 0; rep < 6; ++rep) {          // the first repetitions warm the clocks up
        cudaEventRecord(e0, 0);
        pyr::k_fma_peak<<<ctas, threads>>>(iters, make_float2(0.5f, 0.25f), out);
        cudaEventRecord(e1, 0);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep >= 2 && ms < best) best = ms;
    }
    cudaError_t e = cudaGetLastError();
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    if (e != cudaSuccess) return set_err(PYR_ECUDA, "pyr_measure_fp32_peak: %s", cudaGetErrorString(e));
    const double flops = (double)ctas * threads * (double)iters * 8.0 * 4.0;
    *tflops = (float)(flops / (best * 1e-3) / 1e12);
    if (sm_mhz_effective) *sm_mhz_effective = (float)(flops / (best * 1e-3) / ((double)sms * 128.0 * 2.0) / 1e6);
    return PYR_OK;
}

const char *pyr_kernel_name(int i) { return (i >= 0 && i < 4) ? k_names[i] : ""; }

}  // extern "C"
