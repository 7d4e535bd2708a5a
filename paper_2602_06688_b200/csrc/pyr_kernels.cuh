// pyr_kernels.cuh -- device plan, kernels and their launch geometry (included by pyr.cu for the
// types and by pyr_inst.cu, which instantiates the kernels of ONE transform size per
// translation unit so that the sizes compile in parallel).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include "pyr_fft.cuh"

namespace pyr {

constexpr int RT = 4;   // rows per tile of the intermediate R: one 32-byte sector = RT complex64

// Programmatic dependent launch (PDL): the kernels of one pyr_compute are launched with
// cudaLaunchAttributeProgrammaticStreamSerialization, so a kernel's CTAs may start -- and load their twiddles, set up
// barriers -- while the previous kernel drains; pdl_wait() blocks until that kernel has completed and its writes are
// visible (a no-op for a normally launched kernel), pdl_trigger() lets the next kernel's CTAs be scheduled.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

struct DevPlan {
    int P, N, M, J, B, b, Nd, Nq, o;
    int n_valid;
    int JC, Jc;                // k_cols: j-chunks (blockIdx.z) of Jc distinct y-tilts each
    int KC, Kc;                // k_rows: chunks (blockIdx.y) of Kc tasks each
    const float2 *tw1, *tw2;   // twiddle tables (see Twid)
    const float2 *gx, *gy;     // 1-D masks in digit-reversed register order (custom masks only)
    const float2 *hw1, *hw2;   // twiddle tables of the half-length transform (H = N/2)
    const float2 *lw1, *lw2;   // twiddle tables of the 1024-point one-warp line of the two-halves kernels (= hw1, hw2 at N = 2048)
    const float2 *hx, *hy;     // [M][P], [J][P]  tilt phasor * exp(-2 pi i n / N) / 2 (half-band split)
    const float2 *tx;          // [M][P]  exp(i 2 pi a_kx (x - c_p)/P) / N
    const float2 *ty;          // [J][P]  exp(i 2 pi a_jy (y - c_p)/P) / N
    const int2 *tasks;         // [M]     (y-tilt j, modulation point k) of every point, sorted by j
    int hJC, hJc;              // k_cols_h: j-chunks (blockIdx.z) of hJc distinct y-tilts each
    int TC, Tc;                // k_rows_h: chunks (blockIdx.y) of Tc tasks each
    int SC;                    // chunks of S written by the rows kernel in use (KC or TC; set at launch)
    const unsigned char *valid;  // [Nq][Nq]
    float2 *R;                 // [B][J][N/RT][P][RT]  column-pass result, tiled so that both passes
                               //                      touch whole 32-byte sectors
    float *S;                  // [KC][B][N][Nd]  x-binned partial intensity rows (true coordinates)
    float *partial;            // [B][Nd]         per-detector-row sums over valid pixels
    // general (non-separable) mask path, allocated by pyr_plan_set_mask
    const float2 *MT;          // [N][N]  mask, MT[p][slot(pv)] = mask[v(pv)][u(p)], p / pv = digit-reversed positions
    float2 *F1;                // [B*kch][ceil(P/RT)][N][RT]  x-spectra of the pupil rows (position order)
    float2 *G;                 // [B*kch][N/RT][N][RT]        after forward-y, mask, inverse-y
    int kch;                   // modulation points per chunk of the general path
    float2 *E0;                // [B][NG][P][P]  A exp(i gscale phi), column-contiguous (k_field; N_fft = 2048 only)
    // polychromatic sensor (pyr_plan_create_poly): NG > 1 field groups (wavelengths), the pupil phase of group g is
    // gscale[g] * phase, y-tilt j belongs to group jgroup[j] (consecutive j of a group are contiguous)
    // L2-resident schedule (pyr_plan_set_schedule, N_fft = 2048): the two passes run per chunk of y-tilts; R is a ring
    // of jring y-tilt slots that stays in L2, a launch covers y-tilts [cj0, cj0 + cjn) / tasks [ct0, ct0 + ctn) and the
    // row kernel writes chunk slot cslot of S.  jring == 0: one launch each over everything.
    int jring, cj0, cjn, ct0, ctn, cslot;
    const float2 *gx2, *gy2;   // [2048] 1-D masks in the position order of the two-halves kernels (transform length 2048)
    float2 *E0r;               // [B][NG][P][P]  A exp(i gscale phi), row-contiguous (k_field_r; general masks at length 2048)
    const float2 *w2k;         // [1024] exp(-2 pi i n / 2048): the radix-2 step of the 2048-point general-mask kernels
    int twin;                  // k_rows (table kernels) with the built-in mask: out-of-band rows y', y' + N/2 share one line (6.4)
    int NG;
    const float *gscale;       // [NG] (NULL when there is one group of scale 1: the monochromatic sensor)
    const int *jgroup;         // [J]  (NULL likewise)
};

__device__ __forceinline__ float group_scale(const DevPlan &pd, int j) { return pd.gscale ? __ldg(&pd.gscale[__ldg(&pd.jgroup[j])]) : 1.0f; }

__device__ __forceinline__ size_t r_index(const DevPlan &pd, int s, int j, int yp, int x) {
    return ((((size_t)s * pd.J + j) * (pd.N / RT) + yp / RT) * pd.P + x) * RT + yp % RT;
}

// x-binning of one finished intensity row (NL samples in sf, shared memory) by the TPL threads
// of its group, stored rotated by the pupil offset o at row yt of chunk `chunk` of S; yt2 >= 0:
// the same values also go to row yt2 (the out-of-band twin row of the half-band form).
template <int TPL>
__device__ __forceinline__ void store_binned_row(const DevPlan &pd, const float *sf, int t, int chunk, int s,
                                                 int NL, int yt, int yt2) {
    const int b = pd.b, Nd = pd.Nd, ob = pd.o / b;
    float *__restrict__ Sbase = pd.S + ((size_t)chunk * pd.B + s) * NL * Nd;
    for (int X = t; X < Nd; X += TPL) {
        float sum = 0.f;
        for (int i = 0; i < b; ++i) sum += sf[X * b + i];
        const int Xr = (X + ob) % Nd;
        Sbase[(size_t)yt * Nd + Xr] = sum;
        if (yt2 >= 0) Sbase[(size_t)yt2 * Nd + Xr] = sum;
    }
}

// zeros to rows yt (and yt2 >= 0) of chunk `chunk` of S: a slot of S that a row does not use (k_t2_rows)
template <int TPL>
__device__ __forceinline__ void zero_binned_row(const DevPlan &pd, int t, int chunk, int s, int NL, int yt, int yt2) {
    const int Nd = pd.Nd;
    float *__restrict__ Sbase = pd.S + ((size_t)chunk * pd.B + s) * NL * Nd;
    for (int X = t; X < Nd; X += TPL) {
        Sbase[(size_t)yt * Nd + X] = 0.f;
        if (yt2 >= 0) Sbase[(size_t)yt2 * Nd + X] = 0.f;
    }
}

// ---------------------------------------------------------------- k_cols
// (Table-mask kernels.  Their template parameter N is the TRANSFORM length; pd.N, the logical
// N_fft, is smaller when N_fft is not a power of two: the circulant operator of length pd.N is then
// embedded in a cyclic convolution of length N >= pd.N + P - 1 whose table is built by the plan,
// and only the first pd.N outputs of a line are kept.)
// CTA = G adjacent pupil columns of one source; loops over the distinct y-tilts of its chunk.
// a1 (field build) is the load stage: A exp(i phi) is evaluated once per pixel, kept in
// registers, and multiplied by the y-tilt phasor of every j on the fly.
template <int N, int THREADS, int MINB, int PRUNE>
__global__ void __launch_bounds__(THREADS, MINB)
k_cols(const DevPlan pd, const float *__restrict__ amp, const float *__restrict__ phase) {
    using L = Line<N>;
    constexpr int G = THREADS / L::TPL, NZ = L::N1 / PRUNE;
    extern __shared__ float2 smem[];
    const int g = threadIdx.x / L::TPL, t = threadIdx.x % L::TPL;
    float2 *sm = smem + g * L::SMEM_LINE;
    const int P = pd.P, s = blockIdx.y;
    int x = blockIdx.x * G + g;
    const bool active = x < P;
    if (!active) x = P - 1;
    const int j0 = blockIdx.z * pd.Jc, j1 = min(pd.J, j0 + pd.Jc);
    pdl_trigger();

    Twid<N> tw;
    tw.load(t, pd.tw1, pd.tw2);
    float2 e0[L::B1][NZ];
    auto build_field = [&](float scale) {      // a1: A exp(i scale phi) of this thread's pixels
        // all loads first (the compiler does not move them across the sincosf bodies: one exposed latency each)
#pragma unroll
        for (int i = 0; i < L::B1; ++i)
#pragma unroll
            for (int n1 = 0; n1 < NZ; ++n1) {
                const int y = n1 * L::S1 + t + L::TPL * i;
                const size_t idx = ((size_t)s * P + min(y, P - 1)) * P + x;
                e0[i][n1] = make_float2(__ldg(&amp[idx]), __ldg(&phase[idx]));
            }
#pragma unroll
        for (int i = 0; i < L::B1; ++i)
#pragma unroll
            for (int n1 = 0; n1 < NZ; ++n1) {
                const int y = n1 * L::S1 + t + L::TPL * i;
                float2 e = make_float2(0.f, 0.f);
                if (y < P) {
                    const float a = e0[i][n1].x;
                    float sn, cs;
                    sincosf(scale * e0[i][n1].y, &sn, &cs);
                    e = make_float2(a * cs, a * sn);
                }
                e0[i][n1] = e;
            }
    };
    float cur_scale = j0 < j1 ? group_scale(pd, j0) : 1.0f;
    build_field(cur_scale);
    for (int j = j0; j < j1; ++j) {
        if (pd.NG > 1) {                          // polychromatic: the next wavelength's field
            const float sc = group_scale(pd, j);
            if (sc != cur_scale) { cur_scale = sc; build_field(sc); }
        }
        float2 v[16];
#pragma unroll
        for (int i = 0; i < L::B1; ++i)
#pragma unroll
            for (int n1 = 0; n1 < NZ; ++n1) {
                const int y = n1 * L::S1 + t + L::TPL * i;
                v[i * L::N1 + n1] = y < P ? cmul(e0[i][n1], __ldg(&pd.ty[j * P + y])) : make_float2(0.f, 0.f);
            }
        LineConv<N, PRUNE, false>::run(v, sm, t, g, tw, pd.gy);
        if (active) {
#pragma unroll
            for (int i = 0; i < L::B1; ++i)
#pragma unroll
                for (int n1 = 0; n1 < L::N1; ++n1) {
                    const int yp = n1 * L::S1 + t + L::TPL * i;
                    if (yp < pd.N) pd.R[r_index(pd, s, j, yp, x)] = v[i * L::N1 + n1];   // pd.N < N: embedded size
                }
        }
        // no barrier: the next j first writes exactly the slots this thread read last
    }
}

// ---------------------------------------------------------------- k_rows
// CTA = G adjacent rows y' of one source (G is a multiple of RT or divides it, so a CTA reads
// whole tiles of R); loops over the tasks (j, k) of its chunk; |O_k|^2 accumulates in registers;
// x-binning in the epilogue.
template <int N, int THREADS, int MINB, int PRUNE>
__global__ void __launch_bounds__(THREADS, MINB)
k_rows(const DevPlan pd) {
    using L = Line<N>;
    constexpr int G = THREADS / L::TPL, NZ = L::N1 / PRUNE;
    extern __shared__ float2 smem[];
    const int g = threadIdx.x / L::TPL, t = threadIdx.x % L::TPL;
    float2 *sm = smem + g * L::SMEM_LINE;
    const int P = pd.P;
    const int NL = pd.N;                        // logical N_fft (<= N, the transform length)
    // Built-in mask (pd.twin): rows y' and y' + NL/2 of the y-pass result carry the same intensities outside the band
    // ((y' + NL/4) mod NL/2) < P of the two pupil images (the identity holds for any even NL), so
    // one line serves both: NL/2 + P row tasks per source instead of NL.  Custom masks: every row its own task.
    const int HL = NL / 2, rows = pd.twin ? HL + P : NL;
    const int total = pd.B * rows;
    int task = blockIdx.x * G + g;              // (s, row task)
    const bool active = task < total;
    if (!active) task = total - 1;
    const int rt_ = task % rows, s = task / rows;
    const int yp = !pd.twin || rt_ < HL ? rt_ : HL + (HL / 2 + (rt_ - HL)) % HL;
    const bool dup = pd.twin && rt_ < HL && ((rt_ + HL / 2) % HL) >= P;
    const int i0 = blockIdx.y * pd.Kc, i1 = min(pd.M, i0 + pd.Kc);

    Twid<N> tw;
    tw.load(t, pd.tw1, pd.tw2);
    float acc[16];
#pragma unroll
    for (int e = 0; e < 16; ++e) acc[e] = 0.f;
    pdl_trigger();
    pdl_wait();                                     // R is complete

    for (int it = i0; it < i1; ++it) {
        const int2 tk = pd.tasks[it];              // (y-tilt j, modulation point k)
        float2 v[16];
#pragma unroll
        for (int i = 0; i < L::B1; ++i)
#pragma unroll
            for (int n1 = 0; n1 < NZ; ++n1) {
                const int x = n1 * L::S1 + t + L::TPL * i;
                v[i * L::N1 + n1] = x < P ? cmul(__ldg(&pd.R[r_index(pd, s, tk.x, yp, x)]), __ldg(&pd.tx[tk.y * P + x]))
                                          : make_float2(0.f, 0.f);
            }
        LineConv<N, PRUNE, false>::run(v, sm, t, g, tw, pd.gx);
#pragma unroll
        for (int e = 0; e < 16; ++e) acc[e] += v[e].x * v[e].x + v[e].y * v[e].y;
        // no barrier: the next point first writes exactly the slots this thread read last
    }
    // x-binning through the (now idle) exchange line, then store at the true coordinates
    float *sf = reinterpret_cast<float *>(sm);
    group_sync<L::TPL>(g);
#pragma unroll
    for (int i = 0; i < L::B1; ++i)
#pragma unroll
        for (int n1 = 0; n1 < L::N1; ++n1) sf[n1 * L::S1 + t + L::TPL * i] = acc[i * L::N1 + n1];
    group_sync<L::TPL>(g);
    if (active) store_binned_row<L::TPL>(pd, sf, t, blockIdx.y, s, NL, (yp + pd.o) % NL, dup ? (yp + HL + pd.o) % NL : -1);
}

// ================================================================ half-band split (built-in mask)
// The 1-D pyramid mask g(u) = (-i)^|f(u)| sends the positive frequencies of a line to +N/4 and
// the negative ones to -N/4.  Writing w = exp(-2 pi i / N), H = N/2 and, for a line x supported
// on [0, P), P <= H:
//     z(n)  = x(n) w^n                       (n < H; the twist is folded into the tilt tables)
//     e     = IDFT_H( m . DFT_H(z) ),        m(u) = (-1)^u (u < H/2 ? 1 : -1)      (real signs)
//     q(n)  = +z(n - H/2)  for n >= H/2,     -z(n + H/2)  for n < H/2
// one has, up to a unit factor that depends on n only (and so drops out of every |.|^2 below),
//     (C x)(n) = N ( q(n) + (2/N) e(n) ),    (C x)(n + H) = N ( q(n) - (2/N) e(n) ),   0 <= n < H
// (only the odd harmonics of the difference of the two shifted half-bands survive; derivation
// and the numerical check against the plain definition are in DESIGN.md).  Both passes therefore
// run HALF-length transforms: 0.45x the butterflies and half the shared-memory exchange volume
// of the full-length line operator.  Exact, so parity with the oracle is unchanged.
// Tables hx, hy hold tilt phasor * w^n / 2; the remaining 1/N per axis is the 2/N above.

// k_cols_h: as k_cols (CTA = G pupil columns of one source, loop over its chunk of y-tilts).
template <int H, int E, int THREADS, int MINB, int PRUNE>
__global__ void __launch_bounds__(THREADS, MINB)
k_cols_h(const DevPlan pd, const float *__restrict__ amp, const float *__restrict__ phase) {
    using L = Line<H, E>;
    using LC = LineConv<H, PRUNE, true, E>;
    constexpr int G = THREADS / L::TPL, NZ = L::N1 / PRUNE, N1 = L::N1;
    extern __shared__ float2 smem[];
    const int g = threadIdx.x / L::TPL, t = threadIdx.x % L::TPL;
    float2 *sm = smem + g * L::SMEM_LINE;
    const int P = pd.P, s = blockIdx.y;
    int x = blockIdx.x * G + g;
    const bool active = x < P;
    if (!active) x = P - 1;
    const int j0 = blockIdx.z * pd.hJc, j1 = min(pd.J, j0 + pd.hJc);
    const float c = 1.0f / (float)H;            // 2/N
    pdl_trigger();

    Twid<H, E> tw;
    tw.load(t, pd.hw1, pd.hw2);
    float2 e0[L::B1][NZ];
    auto build_field = [&](float scale) {      // a1: A exp(i scale phi) of this thread's pixels
        // all loads first (the compiler does not move them across the sincosf bodies: one exposed latency each)
#pragma unroll
        for (int i = 0; i < L::B1; ++i)
#pragma unroll
            for (int n1 = 0; n1 < NZ; ++n1) {
                const int y = n1 * L::S1 + t + L::TPL * i;
                const size_t idx = ((size_t)s * P + min(y, P - 1)) * P + x;
                e0[i][n1] = make_float2(__ldg(&amp[idx]), __ldg(&phase[idx]));
            }
#pragma unroll
        for (int i = 0; i < L::B1; ++i)
#pragma unroll
            for (int n1 = 0; n1 < NZ; ++n1) {
                const int y = n1 * L::S1 + t + L::TPL * i;
                float2 e = make_float2(0.f, 0.f);
                if (y < P) {
                    const float a = e0[i][n1].x;
                    float sn, cs;
                    sincosf(scale * e0[i][n1].y, &sn, &cs);
                    e = make_float2(a * cs, a * sn);
                }
                e0[i][n1] = e;
            }
    };
    float cur_scale = j0 < j1 ? group_scale(pd, j0) : 1.0f;
    build_field(cur_scale);
    // Addresses: yp = c + t with c = n1*S1 + TPL*i a multiple of RT, so element (yp, x) of R_j sits
    // at  r0 + j*jstride + (c/RT)*(P*RT)  float2 from R, r0 depending on (s, t, x) only.
    // (tiny transforms whose strides are not multiples of RT take the general index)
    constexpr bool ALIGNED = L::S1 % RT == 0 && L::TPL % RT == 0 && H % RT == 0;
    const size_t jstride = (size_t)(pd.N / RT) * P * RT;
    const size_t rstep = (size_t)P * RT;          // RT rows further
    float2 *const r0 = pd.R + (size_t)s * pd.J * jstride + ((size_t)(t / RT) * P + x) * RT + t % RT;
    const float2 *const hy0 = pd.hy + t;
    // the y-tilt phasors of the NEXT j are fetched while the current line is transformed
    float2 hyn[L::B1][NZ];
    auto fetch_hy = [&](int j) {
        const float2 *hyj = hy0 + (size_t)j * P;
#pragma unroll
        for (int i = 0; i < L::B1; ++i)
#pragma unroll
            for (int n1 = 0; n1 < NZ; ++n1) {
                const int cy = n1 * L::S1 + L::TPL * i;
                hyn[i][n1] = cy + t < P ? __ldg(hyj + cy) : make_float2(0.f, 0.f);
            }
    };
    if (j0 < j1) fetch_hy(j0);
    for (int j = j0; j < j1; ++j) {
        if (pd.NG > 1) {                          // polychromatic: the next wavelength's field
            const float sc = group_scale(pd, j);
            if (sc != cur_scale) { cur_scale = sc; build_field(sc); }
        }
        float2 v[L::EPT], z[L::B1][NZ];
#pragma unroll
        for (int i = 0; i < L::B1; ++i)
#pragma unroll
            for (int n1 = 0; n1 < NZ; ++n1) {
                z[i][n1] = cmul(e0[i][n1], hyn[i][n1]);
                v[i * N1 + n1] = z[i][n1];
            }
        if (j + 1 < j1) fetch_hy(j + 1);
        LC::run(v, sm, t, g, tw, nullptr);
        if (active) {
            float2 *rj = r0 + (size_t)j * jstride;
#pragma unroll
            for (int i = 0; i < L::B1; ++i)
#pragma unroll
                for (int n1 = 0; n1 < N1; ++n1) {
                    const int cy = n1 * L::S1 + L::TPL * i;
                    const int qi = (n1 + N1 / 2) % N1;
                    float2 q = make_float2(0.f, 0.f);
                    if (qi < NZ) q = n1 >= N1 / 2 ? z[i][qi] : make_float2(-z[i][qi].x, -z[i][qi].y);
                    const float2 lo = fma2(bc(c), v[i * N1 + n1], q), hi = fma2(bc(-c), v[i * N1 + n1], q);
                    // out of the band q = 0 and the hi row is minus the lo row: k_rows_h never reads it
                    const bool band = qi < NZ && ((cy + t + H / 2) % H) < P;
                    if (ALIGNED) {
                        rj[(cy / RT) * rstep] = lo;
                        if (band) rj[((cy + H) / RT) * rstep] = hi;
                    } else {
                        pd.R[r_index(pd, s, j, cy + t, x)] = lo;
                        if (band) pd.R[r_index(pd, s, j, cy + t + H, x)] = hi;
                    }
                }
        }
    }
}

// k_rows_h: every group of TPL = H/E threads owns one row y' of R and loops over its chunk of
// tasks (j, k).  Intensities of samples n and n + H accumulate in registers (one
// accumulator where q is identically zero: there both are c^2 |e|^2).  Two tasks per loop iteration, loads of both in
// flight together.  (The one-warp-per-line size, H = 1024, has its own kernels: k_cols_t / k_rows_t below.)
template <int H, int E, int THREADS, int MINB, int PRUNE>
__global__ void __launch_bounds__(THREADS, MINB)
k_rows_h(const DevPlan pd) {
    using L = Line<H, E>;
    using LC = LineConv<H, PRUNE, true, E>;
    constexpr int G = THREADS / L::TPL, NZ = L::N1 / PRUNE, N1 = L::N1, NIN = L::B1 * NZ;
    constexpr int N = 2 * H;
    extern __shared__ float2 smem[];
    const int g = threadIdx.x / L::TPL, t = threadIdx.x % L::TPL;
    float2 *sm = smem + g * L::SMEM_LINE;
    const int P = pd.P, M = pd.M;
    // Rows y' and y' + H of R are q(y') +- c e(y'); where q(y') = 0 -- outside the band
    // ((y' + H/2) mod H) < P of the two pupil images -- they differ by a sign only, their
    // intensities are identical and ONE line serves both output rows.  Row tasks per source:
    // the H "lo" rows (duplicated on store when out of band), then the P in-band "hi" rows.
    const int rows = H + P, total = pd.B * rows;
    int task = blockIdx.x * G + g;              // (s, row task)
    const bool active = task < total;
    if (!active) task = total - 1;
    const int rt_ = task % rows, s = task / rows;
    const int yp = rt_ < H ? rt_ : H + (H / 2 + (rt_ - H)) % H;
    const bool dup = rt_ < H && ((rt_ + H / 2) % H) >= P;
    const int i0 = blockIdx.y * pd.Tc, i1 = min(M, i0 + pd.Tc);
    const float c = 1.0f / (float)H;            // 2/N

    Twid<H, E> tw;
    tw.load(t, pd.hw1, pd.hw2);
    float alo[L::EPT], ahi[L::EPT];
#pragma unroll
    for (int e = 0; e < L::EPT; ++e) alo[e] = ahi[e] = 0.f;
    pdl_trigger();
    pdl_wait();                                     // R is complete

    // |q +- c e|^2 of one finished line into the accumulators
    auto accumulate = [&](const float2 *v, const float2 *z) {
#pragma unroll
        for (int i = 0; i < L::B1; ++i)
#pragma unroll
            for (int n1 = 0; n1 < N1; ++n1) {
                const int e = i * N1 + n1, qi = (n1 + N1 / 2) % N1;
                if (qi < NZ) {
                    const float2 zq = z[i * NZ + qi];
                    const float2 q = n1 >= N1 / 2 ? zq : make_float2(-zq.x, -zq.y);
                    const float2 lo = fma2(bc(c), v[e], q), hi = fma2(bc(-c), v[e], q);
                    alo[e] += lo.x * lo.x + lo.y * lo.y;
                    ahi[e] += hi.x * hi.x + hi.y * hi.y;
                } else {
                    alo[e] += v[e].x * v[e].x + v[e].y * v[e].y;
                }
            }
    };
    // Addresses: x = c + t with c = n1*S1 + TPL*i, so R_j[yp][x] sits at r0 + j*jstride + c*RT and the
    // phasor of point k at hx0 + k*P + c (compile-time c: immediate offsets, no per-element IMAD).
    const size_t jstride = (size_t)(pd.N / RT) * P * RT;
    const float2 *const r0 = pd.R + (size_t)s * pd.J * jstride + ((size_t)(yp / RT) * P + t) * RT + yp % RT;
    const float2 *const hx0 = pd.hx + t;
    // z = (row of R) x (x-tilt phasors) of one task
    auto inputs = [&](int2 tk, float2 *z) {
        const float2 *rj = r0 + (size_t)tk.x * jstride, *xk = hx0 + (size_t)tk.y * P;
#pragma unroll
        for (int i = 0; i < L::B1; ++i)
#pragma unroll
            for (int n1 = 0; n1 < NZ; ++n1) {
                const int cx = n1 * L::S1 + L::TPL * i;
                z[i * NZ + n1] = cx + t < P ? cmul(__ldg(rj + cx * RT), __ldg(xk + cx)) : make_float2(0.f, 0.f);
            }
    };
    auto expand = [&](float2 *v, const float2 *z) {
#pragma unroll
        for (int i = 0; i < L::B1; ++i)
#pragma unroll
            for (int n1 = 0; n1 < NZ; ++n1) v[i * N1 + n1] = z[i * NZ + n1];
    };
    // the inputs of a task into L1 ahead of their use (no registers held)
    auto prefetch = [&](int2 tk) {
        const float2 *rj = r0 + (size_t)tk.x * jstride, *xk = hx0 + (size_t)tk.y * P;
#pragma unroll
        for (int i = 0; i < L::B1; ++i)
#pragma unroll
            for (int n1 = 0; n1 < NZ; ++n1) {
                const int cx = n1 * L::S1 + L::TPL * i;
                if (cx + t < P) {
                    asm volatile("prefetch.global.L1 [%0];" ::"l"(rj + cx * RT));
                    asm volatile("prefetch.global.L1 [%0];" ::"l"(xk + cx));
                }
            }
    };
    // two tasks per iteration: both sets of loads are in flight together; the next pair is prefetched into L1
    // while this pair is transformed
    for (int it = i0; it < i1; it += 2) {
        const bool two = it + 1 < i1;
        float2 v[L::EPT], za[L::B1 * NZ], zb[L::B1 * NZ];
        inputs(pd.tasks[it], za);
        if (two) inputs(pd.tasks[it + 1], zb);
        if (g == 0) {                             // (the G rows of a CTA share their sectors of R and the phasor line)
            if (it + 2 < i1) prefetch(pd.tasks[it + 2]);
            if (it + 3 < i1) prefetch(pd.tasks[it + 3]);
        }
        expand(v, za);
        LC::run(v, sm, t, g, tw, nullptr);
        accumulate(v, za);
        if (two) {
            expand(v, zb);
            LC::run(v, sm, t, g, tw, nullptr);
            accumulate(v, zb);
        }
    }
    // x-binning through the (now idle) exchange line, then store at the true coordinates
    float *sf = reinterpret_cast<float *>(sm);
    group_sync<L::TPL>(g);
#pragma unroll
    for (int i = 0; i < L::B1; ++i)
#pragma unroll
        for (int n1 = 0; n1 < N1; ++n1) {
            const int e = i * N1 + n1, n = n1 * L::S1 + t + L::TPL * i;
            const bool two = (n1 + N1 / 2) % N1 < NZ;
            const float lo = two ? alo[e] : alo[e] * (c * c);
            sf[n] = lo;
            sf[n + H] = two ? ahi[e] : lo;
        }
    group_sync<L::TPL>(g);
    if (active)
        store_binned_row<L::TPL>(pd, sf, t, blockIdx.y, s, N, (yp + pd.o) % N, dup ? (yp + H + pd.o) % N : -1);
}

// ================================================================ N_fft = 2048: row-contiguous R, bulk-copy staging
// (round 2, north_star item (3) "each row or column ... staged in shared memory via TMA")
// For the one-warp-per-line size (H = 1024, E = 32) the intermediate is stored ROW-contiguous,
//     R[s][j][rr][x],  rr < H: row y' = rr ("lo");  rr >= H: the in-band "hi" row y' = H + (H/2 + rr - H) % H,
// i.e. exactly the H + P row tasks of section 6.4, so that the input of a row task is ONE contiguous
// run of P complex64 (3.8 KB) and the G rows of a CTA are one run of G P.  k_rows_t stages them with
// cp.async.bulk (the 1-D TMA bulk copy, completion on an mbarrier; SASS UBLKCP) instead of per-lane 8-byte
// cp.async: two bulk copies per task and CTA (its G rows of R_j, skipped when the next task has the same j;
// the phasor line hx_k, shared by the G lines) replace 64 LDGSTS per lane and their conflicted shared-memory
// writes; the lanes read the staged lines back with conflict-free LDS.64.  k_cols_t transposes its G = 4
// adjacent columns through shared memory and stores whole 32-byte sectors (16 bytes per lane, lane pairs).

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void *src, unsigned bytes, unsigned bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
    unsigned done;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done)
                     : "r"(bar), "r"(parity)
                     : "memory");
    } while (!done);
}

// row task rr of a source -> row y' of the y-pass result, and whether it also serves row y' + H
template <int H>
__device__ __forceinline__ int row_of_task(int rr, int P, bool *dup) {
    *dup = rr < H && ((rr + H / 2) % H) >= P;
    return rr < H ? rr : H + (H / 2 + (rr - H)) % H;
}

// k_cols_t: persistent; a work item is (source, 4 adjacent pupil columns, y-tilt j), item i goes to CTA i mod grid
// (all items cost the same).  A warp owns one column: a = column x of A exp(i phi) (k_field wrote it
// column-contiguous), b = y-tilt line hy_j, both staged by cp.async.bulk into single buffers that are refilled
// for the NEXT item as soon as the product z = a . b sits in registers, i.e. while the line is transformed.
// The 4 warps then write their columns into T [H + P rows][4 columns] in shared memory (32 bytes per row, in the
// 32-byte swizzle of the tensor map: the 16-byte half of a row is exchanged on every other group of four rows, which
// halves the bank conflicts of the column-wise writes) and ONE thread hands T to the TMA: cp.async.bulk.tensor
// stores of 256 rows x 32 bytes into the row-contiguous R (a 3-D tensor map [B J][H + P][2 P floats]; the ragged last
// box and the two-column tail block of a pupil with N_pup % 4 == 2 are clipped by the tensor bounds).  The stores
// are asynchronous: no store instruction, no address arithmetic, and they drain while the next item is transformed
// (measured: 381 MB of R in 32-byte rows at 4.8 TB/s by TMA alone; the 256-bit st.global version of this phase cost
// 0.06 of the kernel's 0.17 ms, section 7 of DESIGN.md).
constexpr int TMA_BOX_ROWS = 256;

__device__ __forceinline__ void tma_store_3d(const CUtensorMap *tm, int c0, int c1, int c2, unsigned src) {
    asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%1, %2, %3}], [%4];" ::"l"(tm), "r"(c0), "r"(c1),
                 "r"(c2), "r"(src)
                 : "memory");
}

// L2 eviction policies for the general-mask passes: the intermediates stream through (evict first), the mask table is
// re-read by every chunk and should stay (evict last)
__device__ __forceinline__ unsigned long long l2_policy_evict_first() {
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ unsigned long long l2_policy_evict_last() {
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void tma_store_3d_hint(const CUtensorMap *tm, int c0, int c1, int c2, unsigned src, unsigned long long pol) {
    asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group.L2::cache_hint [%0, {%1, %2, %3}], [%4], %5;" ::"l"(tm),
                 "r"(c0), "r"(c1), "r"(c2), "r"(src), "l"(pol)
                 : "memory");
}
__device__ __forceinline__ void bulk_g2s_hint(unsigned dst, const void *src, unsigned bytes, unsigned bar, unsigned long long pol) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar), "l"(pol)
                 : "memory");
}
__device__ __forceinline__ float2 ldg_hint(const float2 *p, unsigned long long pol) {
    float2 v;
    asm volatile("ld.global.nc.L2::cache_hint.v2.f32 {%0, %1}, [%2], %3;" : "=f"(v.x), "=f"(v.y) : "l"(p), "l"(pol));
    return v;
}

template <int H, int THREADS, int MINB, int PRUNE>
__global__ void __launch_bounds__(THREADS, MINB)
k_cols_t(const DevPlan pd, const __grid_constant__ CUtensorMap tmR) {
    constexpr int E = 32;
    using L = Line<H, E>;
    using LC = LineConv<H, PRUNE, true, E>;
    constexpr int G = THREADS / 32, N1 = L::N1, NZ = N1 / PRUNE;
    static_assert(L::TPL == 32 && L::B1 == 1 && G == 4, "one warp per line, four columns per CTA");
    extern __shared__ __align__(128) float2 smem[];
    const int g = threadIdx.x >> 5, t = threadIdx.x & 31;
    const int P = pd.P, J = pd.J, rows = H + P;
    const int rpad = (rows + TMA_BOX_ROWS - 1) / TMA_BOX_ROWS * TMA_BOX_ROWS;
    // T [rpad][G] (swizzled, see t_slot) on a 256-byte boundary: the swizzle pattern follows the shared-memory address
    float2 *const Tt = smem + ((256u - (smem_u32(smem) & 255u)) & 255u) / 8u;
    const int WS = L::SMEM_LINE + 2 * P;          // float2 per warp: [exchange line | a | b]
    float2 *const sm = Tt + rpad * G + g * WS;
    float2 *const Ast = sm + L::SMEM_LINE, *const Bst = Ast + P;
    const unsigned bar = smem_u32(Tt + rpad * G + G * WS) + 8 * g;
    const float c = 1.0f / (float)H;              // 2/N
    const int JR = pd.jring ? pd.jring : J;       // y-tilt slots of R
    const int Jn = pd.jring ? pd.cjn : J, Jb = pd.jring ? pd.cj0 : 0;      // y-tilts of this launch
    const int nxb = (P + G - 1) / G, nitems = pd.B * nxb * Jn;
    const unsigned lbytes = (unsigned)P * 8u;
    // float2 slot of (row rr, column g) in T: byte rr * 32 + g * 8 with bit 4 exchanged by bit 7 (CU_TENSOR_MAP_SWIZZLE_32B)
    auto t_slot = [&](int rr) { return rr * G + (g ^ (((rr >> 2) & 1) << 1)); };

    if (t == 0) {
        mbar_init(bar, 1);
        mbar_fence_init();
    }
    __syncwarp();
    Twid<H, E> tw;
    tw.load(t, pd.hw1, pd.hw2);
    pdl_trigger();
    pdl_wait();                                   // E0 (k_field) is complete
    auto issue = [&](int item) {                  // lane 0: stage column x0 + g of source s and the y-tilt line j
        const int xb = item % nxb, rest = item / nxb, j = Jb + rest % Jn, s = rest / Jn, x = min(xb * G + g, P - 1);
        mbar_expect_tx(bar, 2 * lbytes);
        const int grp = pd.NG > 1 ? __ldg(&pd.jgroup[j]) : 0;
        bulk_g2s(smem_u32(Ast), pd.E0 + ((size_t)(s * pd.NG + grp) * P + x) * P, lbytes, bar);
        bulk_g2s(smem_u32(Bst), pd.hy + (size_t)j * P, lbytes, bar);
    };
    int item = blockIdx.x;
    if (t == 0 && item < nitems) issue(item);
    unsigned ph = 0;
    for (; item < nitems; item += gridDim.x, ph ^= 1) {
        const int xb = item % nxb, rest = item / nxb, j = Jb + rest % Jn, s = rest / Jn, x0 = xb * G;
        mbar_wait(bar, ph);
        float2 v[E], z[NZ];
#pragma unroll
        for (int n1 = 0; n1 < NZ; ++n1) {
            z[n1] = n1 * 32 + t < P ? cmul(Ast[n1 * 32 + t], Bst[n1 * 32 + t]) : make_float2(0.f, 0.f);
            v[n1] = z[n1];
        }
        __syncwarp();                              // every lane has its inputs: the buffers can be refilled
        if (t == 0 && item + (int)gridDim.x < nitems) issue(item + gridDim.x);
        LC::run(v, sm, t, g, tw, nullptr);
        // the tensor stores of the previous item have read T (thread 0 issued them), then the CTA meets
        if (threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
        __syncthreads();
#pragma unroll
        for (int n1 = 0; n1 < N1; ++n1) {
            const int yp = n1 * 32 + t, qi = (n1 + N1 / 2) % N1;
            float2 q = make_float2(0.f, 0.f);
            if (qi < NZ) q = n1 >= N1 / 2 ? z[qi] : make_float2(-z[qi].x, -z[qi].y);
            Tt[t_slot(yp)] = fma2(bc(c), v[n1], q);
            // out of the band q = 0 and the hi row is minus the lo row: no row task reads it
            const int bi = (yp + H / 2) % H;
            if (qi < NZ && bi < P) Tt[t_slot(H + bi)] = fma2(bc(-c), v[n1], q);
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // T (generic-proxy writes) before the TMA reads it
        __syncthreads();
        if (threadIdx.x == 0) {
            const int plane = s * JR + j % JR;
            for (int r0 = 0; r0 < rows; r0 += TMA_BOX_ROWS)
                tma_store_3d(&tmR, 2 * x0, r0, plane, smem_u32(Tt + r0 * G));
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        }
        // no barrier here: the next item's transform overlaps the stores; T is protected by the wait above
    }
    if (threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

// k_rows_t: CTA = G warps = G consecutive row tasks of one source; every warp loops over its chunk of tasks (j, k)
// on its own: private exchange line, private double-buffered staging, private mbarriers -- no CTA barrier.
template <int H, int THREADS, int MINB, int PRUNE>
__global__ void __launch_bounds__(THREADS, MINB)
k_rows_t(const DevPlan pd) {
    constexpr int E = 32;
    using L = Line<H, E>;
    using LC = LineConv<H, PRUNE, true, E>;
    constexpr int G = THREADS / 32, N1 = L::N1, NZ = N1 / PRUNE, N = 2 * H;
    static_assert(L::TPL == 32 && L::B1 == 1, "one warp per line");
    extern __shared__ __align__(16) float2 smem[];
    const int g = threadIdx.x >> 5, t = threadIdx.x & 31;
    float2 *sm = smem + g * L::SMEM_LINE;
    const int P = pd.P, M = pd.M, rows = H + P;
    float2 *Rst = smem + G * L::SMEM_LINE + g * (4 * P);   // [2][P]  row of R_j of this warp's row task
    float2 *Xst = Rst + 2 * P;                              // [2][P]  phasor line hx_k
    const unsigned bars = smem_u32(smem + G * L::SMEM_LINE + G * 4 * P) + 16 * g;   // one per stage
    const int nb = (rows + G - 1) / G;
    const int s = blockIdx.x / nb, rr = (blockIdx.x % nb) * G + g;
    const bool active = rr < rows;
    bool dup;
    const int yp = row_of_task<H>(min(rr, rows - 1), P, &dup);
    const int i0 = pd.jring ? pd.ct0 : blockIdx.y * pd.Tc, i1 = pd.jring ? pd.ct0 + pd.ctn : min(M, i0 + pd.Tc);
    const int JR = pd.jring ? pd.jring : pd.J, schunk = pd.jring ? pd.cslot : blockIdx.y;
    const float c = 1.0f / (float)H;              // 2/N

    if (t == 0) {
        mbar_init(bars, 1);
        mbar_init(bars + 8, 1);
        mbar_fence_init();
    }
    __syncwarp();
    const float2 *const Rsrc = pd.R + ((size_t)s * JR * rows + min(rr, rows - 1)) * P;       // + (j mod JR) * rows * P
    const unsigned lbytes = (unsigned)P * 8u;
    // lane 0: stage the inputs of task tk into X stage xst (and its row of R_j into R stage rst when the y-tilt changes)
    auto issue = [&](int2 tk, bool load_r, int rst, int xst) {
        const unsigned bar = bars + 8 * xst;
        mbar_expect_tx(bar, load_r ? 2 * lbytes : lbytes);
        if (load_r) bulk_g2s(smem_u32(Rst + rst * P), Rsrc + (size_t)(tk.x % JR) * rows * P, lbytes, bar);
        bulk_g2s(smem_u32(Xst + xst * P), pd.hx + (size_t)tk.y * P, lbytes, bar);
    };

    Twid<H, E> tw;
    tw.load(t, pd.hw1, pd.hw2);
    float alo[E], ahi[E];
#pragma unroll
    for (int e = 0; e < E; ++e) alo[e] = ahi[e] = 0.f;
    pdl_trigger();
    pdl_wait();                                   // R (k_cols_t) is complete

    int2 tk = i0 < i1 ? pd.tasks[i0] : make_int2(0, 0);
    if (t == 0 && i0 < i1) issue(tk, true, 0, 0);
    int rc = 0;                                   // R stage of the current task
#pragma unroll 1
    for (int it = i0; it < i1; ++it) {
        const int xs = (it - i0) & 1;
        const int2 nx = it + 1 < i1 ? pd.tasks[it + 1] : tk;
        mbar_wait(bars + 8 * xs, ((it - i0) >> 1) & 1);
        const float2 *Rs = Rst + rc * P + t, *Xs = Xst + xs * P + t;
        float2 v[E], za[NZ];
#pragma unroll
        for (int n1 = 0; n1 < NZ; ++n1) {
            za[n1] = n1 * 32 + t < P ? cmul(Rs[n1 * 32], Xs[n1 * 32]) : make_float2(0.f, 0.f);
            v[n1] = za[n1];
        }
        // the stages written next were last read one task ago, before the __syncwarp()s of that line
        const bool newj = nx.x != tk.x;
        if (t == 0 && it + 1 < i1) issue(nx, newj, rc ^ 1, xs ^ 1);
        if (newj) rc ^= 1;
        tk = nx;
        LC::run(v, sm, t, g, tw, nullptr);
#pragma unroll
        for (int n1 = 0; n1 < N1; ++n1) {
            const int qi = (n1 + N1 / 2) % N1;
            if (qi < NZ) {
                const float2 q = n1 >= N1 / 2 ? za[qi] : make_float2(-za[qi].x, -za[qi].y);
                const float2 lo = fma2(bc(c), v[n1], q), hi = fma2(bc(-c), v[n1], q);
                alo[n1] = fmaf(lo.x, lo.x, fmaf(lo.y, lo.y, alo[n1]));
                ahi[n1] = fmaf(hi.x, hi.x, fmaf(hi.y, hi.y, ahi[n1]));
            } else {
                alo[n1] = fmaf(v[n1].x, v[n1].x, fmaf(v[n1].y, v[n1].y, alo[n1]));
            }
        }
    }
    // x-binning through the (now idle) exchange line, then store at the true coordinates
    float *sf = reinterpret_cast<float *>(sm);
    __syncwarp();
#pragma unroll
    for (int n1 = 0; n1 < N1; ++n1) {
        const int n = n1 * 32 + t;
        const bool two = (n1 + N1 / 2) % N1 < NZ;
        const float lo = two ? alo[n1] : alo[n1] * (c * c);
        sf[n] = lo;
        sf[n + H] = two ? ahi[n1] : lo;
    }
    __syncwarp();
    if (active)
        store_binned_row<32>(pd, sf, t, schunk, s, N, (yp + pd.o) % N, dup ? (yp + H + pd.o) % N : -1);
}

// ================================================================ general 2-D mask (pyr_plan_set_mask)
// A mask that is not a product g(v) g(u) (field stop, face or edge defects, other pupil
// separations: SURVEY.md 8(f) f1/f4) takes the three-pass form north_star describes, on the padded
// field with the pupil moved to rows / columns 0..P-1 (the operator is a 2-D circular convolution
// for ANY mask, so the cyclic translation of section 6.2 still holds):
//   k_g_fwd  : forward x-transform of the P non-zero rows (field build fused into the load)
//   k_g_cols : per frequency column: forward y-transform, mask column, inverse y-transform
//   k_g_inv  : inverse x-transform of all N rows, |.|^2 summed over the chunk's points, x-binning
// (As for the table-mask kernels the template parameter N is the transform length; for an N_fft that
// is not a power of two the plan embeds the 2-D circular convolution in one of that length.)
// Spectra stay in the digit-reversed "position" order of LineConv between the passes, so no
// reordering pass exists; F1 and G are tiled like R (RT rows of one column = one 32-byte sector).
// The points are processed in chunks of pd.kch so that G stays a few hundred MB.
__device__ __forceinline__ size_t t_index(int slot, int tiles, int N, int y, int p) {
    return (((size_t)slot * tiles + y / RT) * N + p) * RT + y % RT;
}

template <int N, int THREADS, int MINB, int PRUNE>
__global__ void __launch_bounds__(THREADS, MINB)
k_g_fwd(const DevPlan pd, const float *__restrict__ amp, const float *__restrict__ phase, int i0, int cnt) {
    using L = Line<N>;
    using LC = LineConv<N, PRUNE, false>;
    constexpr int G_ = THREADS / L::TPL, NZ = L::N1 / PRUNE;
    extern __shared__ float2 smem[];
    const int g = threadIdx.x / L::TPL, t = threadIdx.x % L::TPL;
    float2 *sm = smem + g * L::SMEM_LINE;
    const int P = pd.P, PT = (P + RT - 1) / RT;
    const int total = pd.B * cnt * P;
    int line = blockIdx.x * G_ + g;             // (s, kk, y)
    const bool active = line < total;
    if (!active) line = total - 1;
    const int y = line % P, kk = (line / P) % cnt, s = line / (P * cnt);
    const int2 tk = pd.tasks[i0 + kk];          // (j, k)
    Twid<N> tw;
    tw.load(t, pd.tw1, pd.tw2);
    const float2 ty = __ldg(&pd.ty[tk.x * P + y]);
    const float fscale = group_scale(pd, tk.x);
    float2 v[16], xt[L::B1 * NZ];
    // all loads first (the compiler does not move them across the sincosf bodies)
#pragma unroll
    for (int i = 0; i < L::B1; ++i)
#pragma unroll
        for (int n1 = 0; n1 < NZ; ++n1) {
            const int x = min(n1 * L::S1 + t + L::TPL * i, P - 1);
            const size_t idx = ((size_t)s * P + y) * P + x;
            v[i * L::N1 + n1] = make_float2(__ldg(&amp[idx]), __ldg(&phase[idx]));
            xt[i * NZ + n1] = __ldg(&pd.tx[tk.y * P + x]);
        }
#pragma unroll
    for (int i = 0; i < L::B1; ++i)
#pragma unroll
        for (int n1 = 0; n1 < NZ; ++n1) {
            const int x = n1 * L::S1 + t + L::TPL * i;
            float2 e = make_float2(0.f, 0.f);
            if (x < P) {
                const float a = v[i * L::N1 + n1].x;
                float sn, cs;
                sincosf(fscale * v[i * L::N1 + n1].y, &sn, &cs);
                e = cmul(cmul(make_float2(a * cs, a * sn), xt[i * NZ + n1]), ty);
            }
            v[i * L::N1 + n1] = e;
        }
    LC::forward(v, sm, t, g, tw);
    if (active) {
        const int slot = s * cnt + kk;
#pragma unroll
        for (int i = 0; i < L::BL; ++i)
#pragma unroll
            for (int q = 0; q < L::RL; ++q) {
                const int p = (t + L::TPL * i) * L::RL + q;
                pd.F1[t_index(slot, PT, N, y, p)] = v[i * L::RL + q];
            }
    }
}

template <int N, int THREADS, int MINB, int PRUNE>
__global__ void __launch_bounds__(THREADS, MINB)
k_g_cols(const DevPlan pd, int cnt) {
    using L = Line<N>;
    using LC = LineConv<N, PRUNE, false>;
    constexpr int G_ = THREADS / L::TPL, NZ = L::N1 / PRUNE;
    extern __shared__ float2 smem[];
    const int g = threadIdx.x / L::TPL, t = threadIdx.x % L::TPL;
    float2 *sm = smem + g * L::SMEM_LINE;
    const int P = pd.P, PT = (P + RT - 1) / RT;
    const int total = pd.B * cnt * N;
    int line = blockIdx.x * G_ + g;             // (slot, p)
    const bool active = line < total;
    if (!active) line = total - 1;
    const int p = line % N, slot = line / N;
    Twid<N> tw;
    tw.load(t, pd.tw1, pd.tw2);
    float2 v[16];
#pragma unroll
    for (int i = 0; i < L::B1; ++i)
#pragma unroll
        for (int n1 = 0; n1 < NZ; ++n1) {
            const int y = n1 * L::S1 + t + L::TPL * i;
            v[i * L::N1 + n1] = y < P ? __ldg(&pd.F1[t_index(slot, PT, N, y, p)]) : make_float2(0.f, 0.f);
        }
    const float2 *mt = pd.MT + (size_t)p * N;
#pragma unroll
    for (int e = 0; e < 16; ++e)       // the mask column is needed between the two transforms: pull it into L1 now
        asm volatile("prefetch.global.L1 [%0];" ::"l"(mt + e * L::TPL + t));
    LC::run(v, sm, t, g, tw, mt);
    if (active) {
#pragma unroll
        for (int i = 0; i < L::B1; ++i)
#pragma unroll
            for (int n1 = 0; n1 < L::N1; ++n1) {
                const int yp = n1 * L::S1 + t + L::TPL * i;
                if (yp < pd.N) pd.G[t_index(slot, pd.N / RT, N, yp, p)] = v[i * L::N1 + n1];   // pd.N < N: embedded size
            }
    }
}

template <int N, int THREADS, int MINB>
__global__ void __launch_bounds__(THREADS, MINB)
k_g_inv(const DevPlan pd, int cnt, int chunk) {
    using L = Line<N>;
    using LC = LineConv<N, 2, false>;
    constexpr int G_ = THREADS / L::TPL;
    extern __shared__ float2 smem[];
    const int g = threadIdx.x / L::TPL, t = threadIdx.x % L::TPL;
    float2 *sm = smem + g * L::SMEM_LINE;
    const int NL = pd.N;                        // logical N_fft (<= N, the transform length)
    const int total = pd.B * NL;
    int task = blockIdx.x * G_ + g;             // (s, y')
    const bool active = task < total;
    if (!active) task = total - 1;
    const int yp = task % NL, s = task / NL;
    Twid<N> tw;
    tw.load(t, pd.tw1, pd.tw2);
    float acc[16];
#pragma unroll
    for (int e = 0; e < 16; ++e) acc[e] = 0.f;
    for (int kk = 0; kk < cnt; ++kk) {
        const int slot = s * cnt + kk;
        float2 v[16];
#pragma unroll
        for (int i = 0; i < L::BL; ++i)
#pragma unroll
            for (int q = 0; q < L::RL; ++q) {
                const int p = (t + L::TPL * i) * L::RL + q;
                v[i * L::RL + q] = __ldg(&pd.G[t_index(slot, NL / RT, N, yp, p)]);
            }
        LC::inverse(v, sm, t, g, tw);
#pragma unroll
        for (int e = 0; e < 16; ++e) acc[e] += v[e].x * v[e].x + v[e].y * v[e].y;
    }
    float *sf = reinterpret_cast<float *>(sm);
    group_sync<L::TPL>(g);
#pragma unroll
    for (int i = 0; i < L::B1; ++i)
#pragma unroll
        for (int n1 = 0; n1 < L::N1; ++n1) sf[n1 * L::S1 + t + L::TPL * i] = acc[i * L::N1 + n1];
    group_sync<L::TPL>(g);
    if (active) store_binned_row<L::TPL>(pd, sf, t, chunk, s, NL, (yp + pd.o) % NL, -1);
}

// ================================================================ general 2-D mask, transform length 2048 (round 2)
// The three passes above run 128-thread lines with four group barriers per line and are latency-bound at this size
// (profiles/README.md r2: no eligible warp 65-85 %, k_g_inv at 87 % of the L1).  Here a 2048-point transform is two
// 1024-point ones on the one-warp-per-line machinery of k_cols_t / k_rows_t (32 samples per lane, one exchange, only
// __syncwarp), joined by one radix-2 step, w = exp(-2 pi i / 2048):
//   forward (decimation in frequency, x supported on n < 1024):  X[2k] = DFT_1024(x)[k],  X[2k+1] = DFT_1024(x w^n)[k]
//   inverse (decimation in time):  x[n] = E[n] + conj(w^n) O[n],  x[n + 1024] = E[n] - conj(w^n) O[n],
//                                  E = IDFT_1024(X[2k]),  O = IDFT_1024(X[2k+1])
// A spectrum is stored in "position" order u' = (u mod 2) 1024 + u / 2 (the plan permutes the mask accordingly), lane t
// of a warp holding the frequencies k = t + 32 q of either half, so all global and shared accesses are coalesced.
// Intermediates are line-contiguous for their READER and written by TMA tensor stores of 4 lines x 256 elements (as R in
// k_cols_t): F1t[slot][u'][y] (the reader wants a column u' over the P pupil rows), G[slot][y'][u'] (the reader wants a
// row y' over all u'); readers stage whole lines with cp.async.bulk.
struct Gen2Maps { CUtensorMap f1, g; };

template <int PRUNE>
struct Half1024 {
    using L = Line<1024, 32>;
    using LC = LineConv<1024, PRUNE, false, 32>;
    static constexpr int NZ = 32 / PRUNE;
};

// T [rows][4] float2 in the 32-byte swizzle of the tensor maps (see k_cols_t)
__device__ __forceinline__ int t4_slot(int rr, int g) { return rr * 4 + (g ^ (((rr >> 2) & 1) << 1)); }

// pass A: persistent; work item = (slot = (source, point), 4 consecutive pupil rows y), the row block fastest (so that
// neighbouring CTAs write neighbouring 32-byte sectors of F1t at the same time); field build, forward x-transform.
// The TMA stores of an item drain while the next item is built and transformed.
template <int PRUNE>
__global__ void __launch_bounds__(128, 2)
k_h2_fwd(const DevPlan pd, const __grid_constant__ CUtensorMap tmF1, int i0, int cnt) {
    using HC = Half1024<PRUNE>;
    using L = typename HC::L;
    constexpr int NZ = HC::NZ;
    extern __shared__ __align__(128) float2 smem[];
    const int g = threadIdx.x >> 5, t = threadIdx.x & 31;
    float2 *const Tt = smem + ((256u - (smem_u32(smem) & 255u)) & 255u) / 8u;       // [2048][4]
    float2 *const sm = Tt + 2048 * 4 + g * L::SMEM_LINE;
    const int P = pd.P, nyb = (P + 3) / 4, nitems = pd.B * cnt * nyb;
    Twid<1024, 32> tw;
    tw.load(t, pd.lw1, pd.lw2);
    pdl_trigger();
    pdl_wait();
    const unsigned long long pol_stream = l2_policy_evict_first();
    // the field factor A exp(i scale phi) of the NEXT item's row is fetched into registers while the current row is
    // transformed (k_field_r wrote it row-contiguous); the x-tilt line of the point is L1-resident
    float2 xn[NZ];
    auto fetch = [&](int item) {
        const int yb = item % nyb, slot = item / nyb, kk = slot % cnt, s = slot / cnt, y = yb * 4 + g;
        const int grp = pd.NG > 1 ? __ldg(&pd.jgroup[pd.tasks[i0 + kk].x]) : 0;
        const float2 *row = pd.E0r + ((size_t)(s * pd.NG + grp) * P + min(y, P - 1)) * P;
#pragma unroll
        for (int n1 = 0; n1 < NZ; ++n1) xn[n1] = (y < P && n1 * 32 + t < P) ? __ldg(&row[n1 * 32 + t]) : make_float2(0.f, 0.f);
    };
    if ((int)blockIdx.x < nitems) fetch(blockIdx.x);
    for (int item = blockIdx.x; item < nitems; item += gridDim.x) {
        const int yb = item % nyb, slot = item / nyb, kk = slot % cnt;
        const int y = yb * 4 + g;
        const int2 tk = pd.tasks[i0 + kk];          // (j, k)
        float2 x[NZ], v[32];
        const bool on = y < P;
        const float2 ty = on ? __ldg(&pd.ty[tk.x * P + y]) : make_float2(0.f, 0.f);
#pragma unroll
        for (int n1 = 0; n1 < NZ; ++n1) {
            const int n = n1 * 32 + t;
            const float2 e = (on && n < P) ? cmul(cmul(xn[n1], __ldg(&pd.tx[tk.y * P + n])), ty) : make_float2(0.f, 0.f);
            x[n1] = e;
            v[n1] = e;
        }
        if (item + (int)gridDim.x < nitems) fetch(item + gridDim.x);
        HC::LC::forward(v, sm, t, g, tw);            // v[q] = X[2 (t + 32 q)]
        // the tensor stores of the previous item have read T (thread 0 issued them), then the CTA meets
        if (threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
        __syncthreads();
#pragma unroll
        for (int q = 0; q < 32; ++q) Tt[t4_slot(t + 32 * q, g)] = v[q];
#pragma unroll
        for (int n1 = 0; n1 < NZ; ++n1) v[n1] = cmul(x[n1], __ldg(&pd.w2k[n1 * 32 + t]));
        __syncwarp();
        HC::LC::forward(v, sm, t, g, tw);            // v[q] = X[2 (t + 32 q) + 1]
#pragma unroll
        for (int q = 0; q < 32; ++q) Tt[t4_slot(1024 + t + 32 * q, g)] = v[q];
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads();
        if (threadIdx.x == 0) {
            for (int r0 = 0; r0 < 2048; r0 += TMA_BOX_ROWS) tma_store_3d_hint(&tmF1, 2 * yb * 4, r0, slot, smem_u32(Tt + r0 * 4), pol_stream);
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        }
    }
    if (threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

// pass B: persistent; work item = (4 consecutive column positions u', slot), the slot fastest (the CTAs that run at the
// same time share the mask columns in L2): forward y-transform of the P pupil rows, mask column, inverse y-transform
// to all 2048 (logical N) rows.  The next item's column of F1t is staged while the current one is transformed; the TMA
// stores of G drain meanwhile.
// SEP (separable table masks, e.g. the built-in mask at N_fft = 1600 embedded in 2048): the same pass as the column
// pass of the two-pass path -- item = (source, y-tilt j, 4 pupil columns), input = column of E0 (k_field) times the
// y-tilt phasors, mask = the 1-D table gy2, output R[s][j][y'][x].
// HALVES = 1 (SEP only): transform length 1024 (N_fft = 660 embedded in 1024, custom separable masks at N_fft = 1024):
// one 1024-point line operator per column, T has 1024 rows.
template <int PRUNE, bool SEP, int HALVES = 2>
__global__ void __launch_bounds__(128, 2)
k_h2_cols(const DevPlan pd, const __grid_constant__ CUtensorMap tmG, int cnt) {
    static_assert(HALVES == 2 || SEP, "the one-half variant exists for separable masks only");
    constexpr int TROWS = 1024 * HALVES;
    using HC = Half1024<PRUNE>;
    using L = typename HC::L;
    constexpr int NZ = HC::NZ;
    extern __shared__ __align__(128) float2 smem[];
    const int g = threadIdx.x >> 5, t = threadIdx.x & 31;
    float2 *const Tt = smem + ((256u - (smem_u32(smem) & 255u)) & 255u) / 8u;       // [TROWS][4]
    float2 *const sm = Tt + TROWS * 4 + g * L::SMEM_LINE;
    const int P = pd.P, slots = SEP ? pd.B * pd.J : pd.B * cnt, nxb = (P + 3) / 4, nitems = (SEP ? nxb : 512) * slots;
    float2 *const Cst = Tt + TROWS * 4 + 4 * L::SMEM_LINE + g * P;                   // staged column of F1t (SEP: of E0)
    const unsigned bar = smem_u32(Tt + TROWS * 4 + 4 * L::SMEM_LINE + 4 * P) + 8 * g;
    if (t == 0) {
        mbar_init(bar, 1);
        mbar_fence_init();
    }
    __syncwarp();
    Twid<1024, 32> tw;
    tw.load(t, pd.lw1, pd.lw2);
    pdl_trigger();
    pdl_wait();                                   // F1t is complete
    const unsigned long long pol_stream = l2_policy_evict_first(), pol_keep = l2_policy_evict_last();
    auto issue = [&](int item) {                  // lane 0: stage this warp's column of the item
        mbar_expect_tx(bar, (unsigned)P * 8u);
        if (SEP) {
            const int x = min((item % nxb) * 4 + g, P - 1), slot = item / nxb, j = slot % pd.J, s = slot / pd.J;
            const int grp = pd.NG > 1 ? __ldg(&pd.jgroup[j]) : 0;
            bulk_g2s(smem_u32(Cst), pd.E0 + ((size_t)(s * pd.NG + grp) * P + x) * P, (unsigned)P * 8u, bar);
        } else {
            const int slot = item % slots, up = (item / slots) * 4 + g;
            bulk_g2s_hint(smem_u32(Cst), pd.F1 + ((size_t)slot * 2048 + up) * P, (unsigned)P * 8u, bar, pol_stream);
        }
    };
    int item = blockIdx.x;
    if (t == 0 && item < nitems) issue(item);
    unsigned ph = 0;
    for (; item < nitems; item += gridDim.x, ph ^= 1) {
        const int slot = SEP ? item / nxb : item % slots, ub = SEP ? item % nxb : item / slots, up = ub * 4 + g;
        const float2 *__restrict__ mt = SEP ? pd.gy2 : pd.MT + (size_t)up * 2048;
        float2 m[32];
#pragma unroll
        for (int q = 0; q < 32; ++q) m[q] = ldg_hint(&mt[t + 32 * q], pol_keep);      // mask of the even half (coalesced)
        mbar_wait(bar, ph);
        float2 x[NZ], v[32];
#pragma unroll
        for (int n1 = 0; n1 < NZ; ++n1) {
            x[n1] = n1 * 32 + t < P ? Cst[n1 * 32 + t] : make_float2(0.f, 0.f);
            if (SEP && n1 * 32 + t < P) x[n1] = cmul(x[n1], __ldg(&pd.ty[(size_t)(slot % pd.J) * P + n1 * 32 + t]));
            v[n1] = x[n1];
        }
        __syncwarp();                              // every lane has its inputs: the buffer can be refilled
        if (t == 0 && item + (int)gridDim.x < nitems) issue(item + gridDim.x);
        HC::LC::forward(v, sm, t, g, tw);
#pragma unroll
        for (int q = 0; q < 32; ++q) v[q] = cmul(v[q], m[q]);
        HC::LC::inverse(v, sm, t, g, tw);            // E[n1 * 32 + t]
        // the tensor stores of the previous item have read T (thread 0 issued them), then the CTA meets
        if (threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
        __syncthreads();
        if (HALVES == 1) {
#pragma unroll
            for (int q = 0; q < 32; ++q) Tt[t4_slot(q * 32 + t, g)] = v[q];
        } else {
#pragma unroll
            for (int q = 0; q < 32; ++q) {
                Tt[t4_slot(q * 32 + t, g)] = v[q];       // E parks in its rows of T (a lane reads back only what it wrote)
                m[q] = ldg_hint(&mt[1024 + t + 32 * q], pol_keep);     // mask of the odd half
            }
#pragma unroll
            for (int n1 = 0; n1 < NZ; ++n1) v[n1] = cmul(x[n1], __ldg(&pd.w2k[n1 * 32 + t]));
            __syncwarp();
            HC::LC::forward(v, sm, t, g, tw);
#pragma unroll
            for (int q = 0; q < 32; ++q) v[q] = cmul(v[q], m[q]);
            HC::LC::inverse(v, sm, t, g, tw);            // O[n1 * 32 + t]
#pragma unroll
            for (int n1 = 0; n1 < 32; ++n1) {
                const int n = n1 * 32 + t;
                const float2 wo = cmulc(v[n1], __ldg(&pd.w2k[n])), e = Tt[t4_slot(n, g)];
                Tt[t4_slot(n, g)] = cadd(e, wo);
                Tt[t4_slot(n + 1024, g)] = csub(e, wo);
            }
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads();
        if (threadIdx.x == 0) {
            for (int r0 = 0; r0 < pd.N; r0 += TMA_BOX_ROWS) tma_store_3d_hint(&tmG, 2 * ub * 4, r0, slot, smem_u32(Tt + r0 * 4), pol_stream);
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        }
    }
    if (threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

// pass C: one warp per row y' of a source; loops over the points of the chunk: inverse x-transform, |.|^2 accumulated
// in registers, x-binning.  The row of G arrives by two bulk copies (even and odd half of the spectrum); the even
// half's buffer then holds E until the odd half has been transformed.
template <int DUMMY>                              // (a template only so that the header can define it in several translation units)
__global__ void __launch_bounds__(128, 2)
k_h2_inv(const DevPlan pd, int cnt, int chunk) {
    using L = Line<1024, 32>;
    using LC = LineConv<1024, 1, false, 32>;
    extern __shared__ __align__(16) float2 smem[];
    const int g = threadIdx.x >> 5, t = threadIdx.x & 31;
    float2 *const sm = smem + g * L::SMEM_LINE;
    float2 *const Ge = smem + 4 * L::SMEM_LINE + g * 2048, *const Go = Ge + 1024;
    const unsigned bars = smem_u32(smem + 4 * L::SMEM_LINE + 4 * 2048) + 16 * g;
    const int NL = pd.N, total = pd.B * NL;
    int task = blockIdx.x * 4 + g;
    const bool active = task < total;
    if (!active) task = total - 1;
    const int yp = task % NL, s = task / NL;
    if (t == 0) {
        mbar_init(bars, 1);
        mbar_init(bars + 8, 1);
        mbar_fence_init();
    }
    __syncwarp();
    Twid<1024, 32> tw;
    tw.load(t, pd.lw1, pd.lw2);
    float alo[32], ahi[32];
#pragma unroll
    for (int e = 0; e < 32; ++e) alo[e] = ahi[e] = 0.f;
    pdl_trigger();
    pdl_wait();                                   // G is complete
    auto row_of = [&](int kk) { return pd.G + (((size_t)(s * cnt + kk)) * NL + yp) * 2048; };
    const unsigned long long pol_stream = l2_policy_evict_first();
    if (t == 0) {
        mbar_expect_tx(bars, 8192u);
        bulk_g2s_hint(smem_u32(Ge), row_of(0), 8192u, bars, pol_stream);
        mbar_expect_tx(bars + 8, 8192u);
        bulk_g2s_hint(smem_u32(Go), row_of(0) + 1024, 8192u, bars + 8, pol_stream);
    }
#pragma unroll 1
    for (int kk = 0; kk < cnt; ++kk) {
        float2 v[32];
        mbar_wait(bars, kk & 1);
#pragma unroll
        for (int q = 0; q < 32; ++q) v[q] = Ge[t + 32 * q];
        __syncwarp();
        LC::inverse(v, sm, t, g, tw);             // E
#pragma unroll
        for (int n1 = 0; n1 < 32; ++n1) Ge[n1 * 32 + t] = v[n1];     // (a lane reads back only what it wrote)
        mbar_wait(bars + 8, kk & 1);
#pragma unroll
        for (int q = 0; q < 32; ++q) v[q] = Go[t + 32 * q];
        __syncwarp();
        if (t == 0 && kk + 1 < cnt) {              // the odd half is in registers: its buffer can be refilled
            mbar_expect_tx(bars + 8, 8192u);
            bulk_g2s_hint(smem_u32(Go), row_of(kk + 1) + 1024, 8192u, bars + 8, pol_stream);
        }
        LC::inverse(v, sm, t, g, tw);             // O
#pragma unroll
        for (int n1 = 0; n1 < 32; ++n1) {
            const float2 wo = cmulc(v[n1], __ldg(&pd.w2k[n1 * 32 + t])), e = Ge[n1 * 32 + t];
            const float2 lo = cadd(e, wo), hi = csub(e, wo);
            alo[n1] = fmaf(lo.x, lo.x, fmaf(lo.y, lo.y, alo[n1]));
            ahi[n1] = fmaf(hi.x, hi.x, fmaf(hi.y, hi.y, ahi[n1]));
        }
        __syncwarp();
        if (t == 0 && kk + 1 < cnt) {              // E has been read back: the even buffer can be refilled
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            mbar_expect_tx(bars, 8192u);
            bulk_g2s_hint(smem_u32(Ge), row_of(kk + 1), 8192u, bars, pol_stream);
        }
    }
    float *sf = reinterpret_cast<float *>(sm);
    __syncwarp();
#pragma unroll
    for (int n1 = 0; n1 < 32; ++n1) {
        sf[n1 * 32 + t] = alo[n1];
        sf[n1 * 32 + t + 1024] = ahi[n1];
    }
    __syncwarp();
    if (active) store_binned_row<32>(pd, sf, t, chunk, s, NL, (yp + pd.o) % NL, -1);
}

// k_t2_rows: the row pass of the two-pass path for separable TABLE masks at transform lengths 2048 and 1024 (N_fft = 2048 /
// 1024 with a custom separable mask, or N_fft not a power of two embedded: the paper's 24 x 1600 x 1600, 24 x 660 x 660).
// One warp per row task, four consecutive row tasks ("row block") per CTA at a time; the 2048-point line operator is two
// 1024-point halves (see above), the mask table gx2 sits in shared memory, E parks in shared memory while O is
// transformed; inputs (row of R_j, phasor line tx_k) are staged by bulk copies into single buffers that are refilled
// as soon as their product sits in registers.
// PERSISTENT: the (row block, task) pairs, row block slowest, form one sequence of U units that is cut into gridDim.x
// equal ranges, one per CTA -- perfect static balance whatever the shape (with a CTA per (row block, chunk of tasks)
// the paper's 1600 size gave 300 c CTAs on 296 slots: c waves and a sixteen-CTA tail, 19 % of the kernel).  A range
// may start or end inside a row block: the pieces of a row block (at most pd.SC) go to slots 0, 1, ... of S in CTA
// order, and the CTA that holds the last piece writes zeros to the slots that row block does not use, so that k_rebin
// sums pd.SC slots as always.  Twiddles and the mask table are loaded once per CTA.
template <int PRUNE, int HALVES = 2>
__global__ void __launch_bounds__(128, 2)
k_t2_rows(const DevPlan pd) {
    constexpr int TLEN = 1024 * HALVES;           // transform length (HALVES = 1: one 1024-point line operator per task)
    using HC = Half1024<PRUNE>;
    using L = typename HC::L;
    constexpr int NZ = HC::NZ;
    extern __shared__ __align__(16) float2 smem[];
    const int g = threadIdx.x >> 5, t = threadIdx.x & 31;
    const int P = pd.P, NL = pd.N, HL = NL / 2, M = pd.M;
    float2 *const sm = smem + g * L::SMEM_LINE;
    float2 *const Ep = smem + 4 * L::SMEM_LINE + g * 1024;                        // parked E (HALVES = 2)
    float2 *const gxs = smem + 4 * L::SMEM_LINE + (HALVES == 2 ? 4 * 1024 : 0);   // [TLEN] mask table
    float2 *const Rst = gxs + TLEN + g * 2 * P, *const Xst = Rst + P;
    const unsigned bar = smem_u32(gxs + TLEN + 8 * P) + 8 * g;
    const int rows = pd.twin ? HL + P : NL, total = pd.B * rows, nrb = (total + 3) / 4;
    const long long U = (long long)nrb * M, grid = gridDim.x;
    const long long u0 = (long long)blockIdx.x * U / grid, u1 = ((long long)blockIdx.x + 1) * U / grid;
    int rb = (int)(u0 / M), i0 = (int)(u0 - (long long)rb * M), left = (int)(u1 - u0);     // (32-bit loop state)
    if (t == 0) {
        mbar_init(bar, 1);
        mbar_fence_init();
    }
    for (int i = threadIdx.x; i < TLEN; i += 128) gxs[i] = __ldg(&pd.gx2[i]);
    __syncthreads();
    Twid<1024, 32> tw;
    tw.load(t, pd.lw1, pd.lw2);
    pdl_trigger();
    pdl_wait();                                   // R is complete
    const unsigned lbytes = (unsigned)P * 8u;
    unsigned nwait = 0;                           // completed phases of this warp's barrier
    float *const sf = reinterpret_cast<float *>(sm);
#pragma unroll 1
    while (left > 0) {
        const int i1 = min(M, i0 + left);
        int task = rb * 4 + g;
        const bool active = task < total;
        if (!active) task = total - 1;
        const int rt_ = task % rows, s = task / rows;
        const int yp = !pd.twin || rt_ < HL ? rt_ : HL + (HL / 2 + (rt_ - HL)) % HL;
        const bool dup = pd.twin && rt_ < HL && ((rt_ + HL / 2) % HL) >= P;
        const float2 *const Rrow = pd.R + ((size_t)s * pd.J * NL + yp) * P;             // + j NL P
        auto issue = [&](int2 tk, bool load_r) {      // lane 0
            mbar_expect_tx(bar, load_r ? 2 * lbytes : lbytes);
            if (load_r) bulk_g2s(smem_u32(Rst), Rrow + (size_t)tk.x * NL * P, lbytes, bar);
            bulk_g2s(smem_u32(Xst), pd.tx + (size_t)tk.y * P, lbytes, bar);
        };
        float alo[32], ahi[32];
#pragma unroll
        for (int e = 0; e < 32; ++e) alo[e] = ahi[e] = 0.f;
        int2 tk = pd.tasks[i0];
        if (t == 0) issue(tk, true);
#pragma unroll 1
        for (int it = i0; it < i1; ++it) {
            const int2 nx = it + 1 < i1 ? pd.tasks[it + 1] : tk;
            mbar_wait(bar, nwait & 1);
            ++nwait;
            float2 x[NZ], v[32];
#pragma unroll
            for (int n1 = 0; n1 < NZ; ++n1) {
                x[n1] = n1 * 32 + t < P ? cmul(Rst[n1 * 32 + t], Xst[n1 * 32 + t]) : make_float2(0.f, 0.f);   // (R_j stays staged while j does)
                v[n1] = x[n1];
            }
            __syncwarp();                              // the staged lines are in registers: refill
            if (t == 0 && it + 1 < i1) issue(nx, nx.x != tk.x);
            tk = nx;
            HC::LC::forward(v, sm, t, g, tw);
#pragma unroll
            for (int q = 0; q < 32; ++q) v[q] = cmul(v[q], gxs[t + 32 * q]);
            HC::LC::inverse(v, sm, t, g, tw);            // E
            if (HALVES == 1) {
#pragma unroll
                for (int n1 = 0; n1 < 32; ++n1) alo[n1] = fmaf(v[n1].x, v[n1].x, fmaf(v[n1].y, v[n1].y, alo[n1]));
            } else {
#pragma unroll
                for (int n1 = 0; n1 < 32; ++n1) Ep[n1 * 32 + t] = v[n1];
#pragma unroll
                for (int n1 = 0; n1 < NZ; ++n1) v[n1] = cmul(x[n1], __ldg(&pd.w2k[n1 * 32 + t]));
                __syncwarp();
                HC::LC::forward(v, sm, t, g, tw);
#pragma unroll
                for (int q = 0; q < 32; ++q) v[q] = cmul(v[q], gxs[1024 + t + 32 * q]);
                HC::LC::inverse(v, sm, t, g, tw);            // O
#pragma unroll
                for (int n1 = 0; n1 < 32; ++n1) {
                    const float2 wo = cmulc(v[n1], __ldg(&pd.w2k[n1 * 32 + t])), e = Ep[n1 * 32 + t];
                    const float2 lo = cadd(e, wo), hi = csub(e, wo);
                    alo[n1] = fmaf(lo.x, lo.x, fmaf(lo.y, lo.y, alo[n1]));
                    ahi[n1] = fmaf(hi.x, hi.x, fmaf(hi.y, hi.y, ahi[n1]));
                }
            }
            __syncwarp();
        }
        // x-binning through the (now idle) exchange line, then store at the true coordinates into this piece's slot of S
        __syncwarp();
#pragma unroll
        for (int n1 = 0; n1 < 32; ++n1) {
            sf[n1 * 32 + t] = alo[n1];
            if (HALVES == 2) sf[n1 * 32 + t + 1024] = ahi[n1];
        }
        __syncwarp();
        // the pieces of row block rb: CTAs i_first .. i_last (the CTAs whose ranges hold its first and last unit)
        const long long ub = (long long)rb * M;
        const int i_first = (int)(((ub + 1) * grid - 1) / U), i_last = (int)(((ub + M) * grid - 1) / U);
        const int piece = (int)blockIdx.x - i_first;
        const int yt = (yp + pd.o) % NL, yt2 = dup ? (yp + HL + pd.o) % NL : -1;
        if (active) {
            store_binned_row<32>(pd, sf, t, piece, s, NL, yt, yt2);
            if ((int)blockIdx.x == i_last)
                for (int slot = piece + 1; slot < pd.SC; ++slot) zero_binned_row<32>(pd, t, slot, s, NL, yt, yt2);
        }
        __syncwarp();                              // sf is the exchange line of the next row block's transforms
        left -= i1 - i0;
        ++rb;
        i0 = 0;
    }
}

// ---------------------------------------------------------------- test-only: the bare line operator
template <int N, int THREADS, int PRUNE>
__global__ void __launch_bounds__(THREADS)
k_test_line(const DevPlan pd, const float2 *__restrict__ in, float2 *__restrict__ out, int nlines) {
    using L = Line<N>;
    constexpr int G = THREADS / L::TPL, NZ = L::N1 / PRUNE;
    extern __shared__ float2 smem[];
    const int g = threadIdx.x / L::TPL, t = threadIdx.x % L::TPL;
    float2 *sm = smem + g * L::SMEM_LINE;
    int task = blockIdx.x * G + g;
    const bool active = task < nlines;
    if (!active) task = nlines - 1;
    Twid<N> tw;
    tw.load(t, pd.tw1, pd.tw2);
    float2 v[16];
#pragma unroll
    for (int i = 0; i < L::B1; ++i)
#pragma unroll
        for (int n1 = 0; n1 < NZ; ++n1) {
            const int x = n1 * L::S1 + t + L::TPL * i;
            v[i * L::N1 + n1] = x < pd.P ? in[(size_t)task * pd.P + x] : make_float2(0.f, 0.f);
        }
    LineConv<N, PRUNE, false>::run(v, sm, t, g, tw, pd.gx);
    const float sc = 1.0f / (float)pd.N;
    if (active) {
#pragma unroll
        for (int i = 0; i < L::B1; ++i)
#pragma unroll
            for (int n1 = 0; n1 < L::N1; ++n1) {
                const int x = n1 * L::S1 + t + L::TPL * i;
                if (x < pd.N) out[(size_t)task * pd.N + x] = make_float2(v[i * L::N1 + n1].x * sc, v[i * L::N1 + n1].y * sc);
            }
    }
}

// test-only: the line operator in its half-band form, with the unit factor -i exp(+2 pi i n / N)
// that the production kernels drop put back, so that out = (C x) / N as for k_test_line.
template <int H, int E, int THREADS, int PRUNE>
__global__ void __launch_bounds__(THREADS)
k_test_line_h(const DevPlan pd, const float2 *__restrict__ in, float2 *__restrict__ out, int nlines) {
    using L = Line<H, E>;
    constexpr int G = THREADS / L::TPL, NZ = L::N1 / PRUNE, N1 = L::N1, N = 2 * H;
    extern __shared__ float2 smem[];
    const int g = threadIdx.x / L::TPL, t = threadIdx.x % L::TPL;
    float2 *sm = smem + g * L::SMEM_LINE;
    int task = blockIdx.x * G + g;
    const bool active = task < nlines;
    if (!active) task = nlines - 1;
    Twid<H, E> tw;
    tw.load(t, pd.hw1, pd.hw2);
    float2 v[L::EPT], z[L::B1][NZ];
#pragma unroll
    for (int i = 0; i < L::B1; ++i)
#pragma unroll
        for (int n1 = 0; n1 < NZ; ++n1) {
            const int x = n1 * L::S1 + t + L::TPL * i;
            float2 a = make_float2(0.f, 0.f);
            if (x < pd.P) {
                float sn, cs;
                sincospif(-2.0f * (float)x / (float)N, &sn, &cs);
                a = cmul(in[(size_t)task * pd.P + x], make_float2(0.5f * cs, 0.5f * sn));
            }
            z[i][n1] = a;
            v[i * N1 + n1] = a;
        }
    LineConv<H, PRUNE, true, E>::run(v, sm, t, g, tw, nullptr);
    const float c = 1.0f / (float)H;
    if (active) {
#pragma unroll
        for (int i = 0; i < L::B1; ++i)
#pragma unroll
            for (int n1 = 0; n1 < N1; ++n1) {
                const int n = n1 * L::S1 + t + L::TPL * i;
                const int qi = (n1 + N1 / 2) % N1;
                float2 q = make_float2(0.f, 0.f);
                if (qi < NZ) q = n1 >= N1 / 2 ? z[i][qi] : make_float2(-z[i][qi].x, -z[i][qi].y);
                float sn, cs;
                sincospif(2.0f * (float)n / (float)N, &sn, &cs);
                const float2 f = make_float2(sn, -cs);      // -i exp(+2 pi i n / N)
                out[(size_t)task * N + n] = cmul(fma2(bc(c), v[i * N1 + n1], q), f);
                out[(size_t)task * N + n + H] = cmul(fma2(bc(-c), v[i * N1 + n1], q), f);
            }
    }
}

}  // namespace pyr

using pyr::DevPlan;

// Full-length, table-mask kernels (custom separable masks, and N = 16) and their launch geometry.
struct KernelSet {
    void (*cols)(const DevPlan, const float *, const float *);
    void (*rows)(const DevPlan);
    void (*gfwd)(const DevPlan, const float *, const float *, int, int);   // general-mask path
    void (*gcols)(const DevPlan, int);
    void (*ginv)(const DevPlan, int, int);
    void (*test)(const DevPlan, const float2 *, float2 *, int);
    int cols_threads, cols_G, rows_threads, rows_G, test_threads, test_G;
    size_t cols_smem, rows_smem, test_smem;
};

// The half-band-split kernels (built-in mask, N >= 32) and their launch geometry.
struct HalfSet {
    void (*cols)(const DevPlan, const float *, const float *);
    void (*cols_t)(const DevPlan, const CUtensorMap);      // rowmajor: k_cols_t (reads E0, stores R through the tensor map)
    void (*rows)(const DevPlan);
    void (*test)(const DevPlan, const float2 *, float2 *, int);
    int cols_threads, cols_G, rows_threads, rows_G, test_threads, test_G;
    size_t cols_smem, rows_smem, test_smem;
    int N1, N2, N3;                 // factorisation of the half-length transform (twiddle tables)
    bool rowmajor;                  // R is [B][J][H + P][P] (k_cols_t / k_rows_t) instead of the RT-row tiles
    size_t cols_smem_perP, rows_smem_perP;   // dynamic shared memory grows with N_pup (staged lines)
};

struct Gen2Set {
    void (*fwd)(const DevPlan, const CUtensorMap, int, int);
    void (*cols)(const DevPlan, const CUtensorMap, int);
    void (*inv)(const DevPlan, int, int);
    void (*cols_sep)(const DevPlan, const CUtensorMap, int);     // separable table masks: the two-pass path at length 2048
    void (*rows_sep)(const DevPlan);
    void (*cols_sep1)(const DevPlan, const CUtensorMap, int);    // ... at length 1024
    void (*rows_sep1)(const DevPlan);
    size_t fwd_smem, cols_smem_base, inv_smem;     // cols: + 4 P complex (staged columns)
    size_t rows_sep_smem_base, cols_sep1_smem_base, rows_sep1_smem_base;
};

template <int PRUNE>
Gen2Set make_gen2() {
    using L = pyr::Line<1024, 32>;
    Gen2Set k;
    k.fwd = pyr::k_h2_fwd<PRUNE>;
    k.cols = pyr::k_h2_cols<PRUNE, false>;
    k.cols_sep = pyr::k_h2_cols<PRUNE, true>;
    k.rows_sep = pyr::k_t2_rows<PRUNE>;
    k.rows_sep_smem_base = (size_t)(4 * L::SMEM_LINE + 4 * 1024 + 2048) * sizeof(float2) + 4 * 8;   // + 8 P complex (staged lines)
    k.cols_sep1 = pyr::k_h2_cols<PRUNE, true, 1>;
    k.rows_sep1 = pyr::k_t2_rows<PRUNE, 1>;
    k.cols_sep1_smem_base = (size_t)(1024 * 4 + 4 * L::SMEM_LINE) * sizeof(float2) + 4 * 8 + 256;
    k.rows_sep1_smem_base = (size_t)(4 * L::SMEM_LINE + 1024) * sizeof(float2) + 4 * 8;
    k.inv = pyr::k_h2_inv<0>;
    k.fwd_smem = (size_t)(2048 * 4 + 4 * L::SMEM_LINE) * sizeof(float2) + 256;
    k.cols_smem_base = (size_t)(2048 * 4 + 4 * L::SMEM_LINE) * sizeof(float2) + 4 * 8 + 256;
    k.inv_smem = (size_t)(4 * L::SMEM_LINE + 4 * 2048) * sizeof(float2) + 4 * 16;
    return k;
}
Gen2Set pyr_pick_gen2(int prune);      // defined in the N_fft = 2048 translation unit

// Launch geometry per N: threads per CTA and min CTAs/SM (register budget) of k_cols and k_rows.
template <int N> struct Geo { static constexpr int CT = 256, CMINB = 2, RTH = 256, RMINB = 2; };
template <> struct Geo<2048> { static constexpr int CT = 512, CMINB = 1, RTH = 512, RMINB = 1; };

template <int N, int PRUNE>
KernelSet make_set() {
    using L = pyr::Line<N>;
    using G = Geo<N>;
    constexpr int TT = L::TPL > 256 ? L::TPL : 256;
    KernelSet k;
    k.cols = pyr::k_cols<N, G::CT, G::CMINB, PRUNE>;
    k.rows = pyr::k_rows<N, G::RTH, G::RMINB, PRUNE>;
    k.test = pyr::k_test_line<N, TT, PRUNE>;
    k.gfwd = pyr::k_g_fwd<N, G::RTH, G::RMINB, PRUNE>;
    k.gcols = pyr::k_g_cols<N, G::RTH, G::RMINB, PRUNE>;
    k.ginv = pyr::k_g_inv<N, G::RTH, G::RMINB>;
    k.cols_threads = G::CT;  k.cols_G = G::CT / L::TPL;  k.cols_smem = (size_t)k.cols_G * L::SMEM_LINE * sizeof(float2);
    k.rows_threads = G::RTH; k.rows_G = G::RTH / L::TPL; k.rows_smem = (size_t)k.rows_G * L::SMEM_LINE * sizeof(float2);
    k.test_threads = TT;     k.test_G = TT / L::TPL;     k.test_smem = (size_t)k.test_G * L::SMEM_LINE * sizeof(float2);
    return k;
}

template <int N>
KernelSet pick_set(int prune) {
    return prune == 4 ? make_set<N, 4>() : make_set<N, 2>();
}

// Launch geometry of the half-band-split kernels: {samples per thread, threads and min CTAs/SM
// of k_cols_h, of k_rows_h}, chosen from B200 measurements (profiles/README.md):
// H = 1024 (the ELT-scale size): one warp per line, 32 samples per thread (two passes, one exchange
// per transform), 4 rows = one tile of R per CTA; every other size: 16 samples per thread, one
// 64-thread CTA, 8 per SM.
template <int H, int E, int PRUNE, int CT, int CMINB, int RTH, int RMINB>
HalfSet make_half() {
    using L = pyr::Line<H, E>;
    constexpr int CTT = CT > L::TPL ? CT : L::TPL, RTT = RTH > L::TPL ? RTH : L::TPL;
    constexpr int TT = L::TPL > 256 ? L::TPL : 256;
    HalfSet k;
    k.cols = pyr::k_cols_h<H, E, CTT, CMINB, PRUNE>;
    k.rows = pyr::k_rows_h<H, E, RTT, RMINB, PRUNE>;
    k.test = pyr::k_test_line_h<H, E, TT, PRUNE>;
    k.N1 = L::N1; k.N2 = L::N2; k.N3 = L::N3;
    k.rowmajor = false; k.cols_smem_perP = k.rows_smem_perP = 0; k.cols_t = nullptr;
    k.cols_threads = CTT; k.cols_G = CTT / L::TPL; k.cols_smem = (size_t)k.cols_G * L::SMEM_LINE * sizeof(float2);
    k.rows_threads = RTT; k.rows_G = RTT / L::TPL;
    k.rows_smem = (size_t)k.rows_G * L::SMEM_LINE * sizeof(float2);
    k.test_threads = TT;  k.test_G = TT / L::TPL;  k.test_smem = (size_t)k.test_G * L::SMEM_LINE * sizeof(float2);
    return k;
}

// H = 1024: row-contiguous R, four lines per CTA, bulk-copy staging (k_cols_t / k_rows_t)
template <int H, int PRUNE>
HalfSet make_half_t() {
    using L = pyr::Line<H, 32>;
    constexpr int TH = 128, G = TH / 32, TT = 256;
    HalfSet k;
    k.cols = nullptr;
    k.cols_t = pyr::k_cols_t<H, TH, 2, PRUNE>;
    constexpr int RTH = TH, RG = RTH / 32;
    k.rows = pyr::k_rows_t<H, RTH, 2, PRUNE>;
    k.test = pyr::k_test_line_h<H, 32, TT, PRUNE>;
    k.N1 = L::N1; k.N2 = L::N2; k.N3 = L::N3;
    k.rowmajor = true;
    k.cols_threads = TH; k.cols_G = G;
    // T [ceil((H + P) / 256) 256 rows][G] + per warp [exchange line | a | b] + barriers; the plan adds the P-dependent part
    k.cols_smem = (size_t)G * L::SMEM_LINE * sizeof(float2) + G * 8 + 256;
    k.cols_smem_perP = (size_t)2 * G * sizeof(float2);
    k.rows_threads = RTH; k.rows_G = RG;
    k.rows_smem = (size_t)RG * L::SMEM_LINE * sizeof(float2) + RG * 16;      // + 4 G P complex (staged lines)
    k.rows_smem_perP = (size_t)4 * RG * sizeof(float2);
    k.test_threads = TT;  k.test_G = TT / L::TPL;  k.test_smem = (size_t)k.test_G * L::SMEM_LINE * sizeof(float2);
    return k;
}

// Resident 64-thread CTAs per SM asked of ptxas (launch bounds) for the 16-samples-per-thread kernels.  Unpruned
// first butterflies (PRUNE = 1: P > N/4) hold 16 staged inputs more and spill at 128 registers (8 CTAs); measured
// on C2 / C3 (80/256/24, 160/512/48): 8: 44.5 / 64.5 us, 6: 41.0 / 56.8 us, 4: 38.9 / 61.5 us.
template <int H, int PRUNE>
constexpr int half_minb() { return PRUNE == 1 ? (H <= 128 ? 4 : 6) : 8; }
template <int H, int PRUNE>
HalfSet pick_half() {
    if constexpr (H == 1024) return make_half_t<H, PRUNE>();
    else {
        constexpr int MB = half_minb<H, PRUNE>();
        return make_half<H, 16, PRUNE, 64, MB, 64, MB>();
    }
}

template <int H>
HalfSet pick_half_prune(int prune) {
    if (prune == 4) return pick_half<H, 4>();
    if (prune == 2) return pick_half<H, 2>();
    return pick_half<H, 1>();
}

// One translation unit per size (pyr_inst.cu, -DPYR_INST_N=<N>) defines these.
#define PYR_DECLARE_SIZE(N_)                          \
    KernelSet pyr_pick_set_##N_(int prune);           \
    HalfSet pyr_pick_half_##N_(int prune);
PYR_DECLARE_SIZE(16) PYR_DECLARE_SIZE(32) PYR_DECLARE_SIZE(64) PYR_DECLARE_SIZE(128)
PYR_DECLARE_SIZE(256) PYR_DECLARE_SIZE(512) PYR_DECLARE_SIZE(1024) PYR_DECLARE_SIZE(2048)
