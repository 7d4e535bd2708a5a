// chain.cu -- the steps either side of the wavefront sensor (include/chain.h; DESIGN.md
// section 14): on-device phase source (AtmoEvolution + AtmoPropagation), detector model (CCD), pupil-map
// calibrator (PyrPupdataCalibrator) and modal reconstructor (Modalrec).  All four are bound by HBM / L2 traffic or
// by launch latency, none is a large contraction (Modalrec is a mat-vec with B <= a few right-hand sides:
// B/2 flop per byte of R), so they are plain coalesced streaming kernels with grids sized to the SM count.
//
// The CCD noise model is reproducible bit for bit: Philox4x32-10 integer streams, and every float32 step that
// decides an integer written with round-to-nearest intrinsics (__fmaf_rn, __fmul_rn, __fadd_rn, __fdiv_rn,
// __fsqrt_rn, rintf), which nvcc neither fuses nor re-associates; exp / log / cos are short polynomials of
// those (reading C5).
#include <cuda_runtime.h>

#include <cmath>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/chain.h"

namespace {

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

bool on_device(int device, const char *who) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != device) {
        set_err(1, "%s: the plan was created on device %d, the current device is %d", who, device, dev);
        return false;
    }
    return true;
}

int sm_count() {
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    return sms;
}

// ================================================================ atmosphere
constexpr int ATMO_MAX = 128;      // layers x sources per call (kernel parameter space)
struct AtmoShift { int iy, ix; float fy, fx; };
struct AtmoArgs {
    int L, S, P, B, vec;
    float w[16];                   // layer weights (L <= 16 kept by value; more layers: see w_dev)
    AtmoShift sh[ATMO_MAX];        // [B][L]
};

// One thread per four consecutive output pixels of a row (one 16-byte store when N_pup is a multiple of 4 and the
// output is 16-byte aligned; the five samples per screen row that they interpolate between are read through L1:
// neighbouring threads share sectors, so every screen byte is fetched from L2 once per row pair), lanes along x.
__global__ void __launch_bounds__(128) k_atmo(const AtmoArgs a, const float *__restrict__ screens, const float *__restrict__ w_dev,
                                              float *__restrict__ out) {
    const int P = a.P, S = a.S, L = a.L;
    const int x0 = (blockIdx.x * blockDim.x + threadIdx.x) * 4, y = blockIdx.y, b = blockIdx.z;
    if (x0 >= P) return;
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
    for (int l = 0; l < L; ++l) {
        const AtmoShift s = a.sh[b * L + l];
        const float *__restrict__ scr = screens + (size_t)l * S * S;
        const int i = (y + s.iy) % S, i1 = i + 1 == S ? 0 : i + 1;
        const float *__restrict__ r0 = scr + (size_t)i * S, *__restrict__ r1 = scr + (size_t)i1 * S;
        int j = (x0 + s.ix) % S;
        float t[5], u[5];
#pragma unroll
        for (int q = 0; q < 5; ++q) {
            t[q] = __ldg(&r0[j]);
            u[q] = __ldg(&r1[j]);
            j = j + 1 == S ? 0 : j + 1;
        }
        const float w = L <= 16 ? a.w[l] : __ldg(&w_dev[l]);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const float top = fmaf(s.fx, t[q + 1] - t[q], t[q]), bot = fmaf(s.fx, u[q + 1] - u[q], u[q]);
            acc[q] = fmaf(w, fmaf(s.fy, bot - top, top), acc[q]);
        }
    }
    float *__restrict__ o = out + ((size_t)b * P + y) * P + x0;
    if (a.vec) {                                  // N_pup a multiple of 4 and out_phase on a 16-byte boundary
        *reinterpret_cast<float4 *>(o) = make_float4(acc[0], acc[1], acc[2], acc[3]);
    } else {
#pragma unroll
        for (int q = 0; q < 4; ++q)
            if (x0 + q < P) o[q] = acc[q];
    }
}

// ================================================================ CCD noise model (float32, IEEE-exact steps)
__device__ __forceinline__ void philox4x32_10(unsigned c0, unsigned c1, unsigned c2, unsigned c3, unsigned k0, unsigned k1,
                                              unsigned (&o)[4]) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        if (r) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
        const unsigned hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const unsigned hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const unsigned n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    }
    o[0] = c0; o[1] = c1; o[2] = c2; o[3] = c3;
}

__device__ __forceinline__ float u01(unsigned x) { return __fmul_rn(__fadd_rn((float)(x >> 9), 0.5f), 1.1920928955078125e-7f); }

__device__ __forceinline__ float exp_neg(float lam) {
    const float x = -lam;
    const float k = rintf(__fmul_rn(x, 1.44269504088896341f));
    float r = __fmaf_rn(k, -0.693359375f, x);
    r = __fmaf_rn(k, 2.12194440e-4f, r);
    float p = 1.9875691500e-4f;
    p = __fmaf_rn(p, r, 1.3981999507e-3f);
    p = __fmaf_rn(p, r, 8.3334519073e-3f);
    p = __fmaf_rn(p, r, 4.1665795894e-2f);
    p = __fmaf_rn(p, r, 1.6666665459e-1f);
    p = __fmaf_rn(p, r, 5.0000001201e-1f);
    const float r2 = __fmul_rn(r, r);
    float y = __fmaf_rn(p, r2, r);
    y = __fadd_rn(y, 1.0f);
    return __fmul_rn(y, __uint_as_float((unsigned)((int)k + 127) << 23));
}

__device__ __forceinline__ float log01(float u) {
    const unsigned b = __float_as_uint(u);
    int e = (int)((b >> 23) & 0xffu) - 126;
    float x = __uint_as_float((b & 0x007fffffu) | 0x3f000000u);
    if (x < 0.707106781186547524f) { e -= 1; x = __fadd_rn(__fadd_rn(x, x), -1.0f); } else { x = __fadd_rn(x, -1.0f); }
    const float z = __fmul_rn(x, x);
    float y = 7.0376836292e-2f;
    y = __fmaf_rn(y, x, -1.1514610310e-1f);
    y = __fmaf_rn(y, x, 1.1676998740e-1f);
    y = __fmaf_rn(y, x, -1.2420140846e-1f);
    y = __fmaf_rn(y, x, 1.4249322787e-1f);
    y = __fmaf_rn(y, x, -1.6668057665e-1f);
    y = __fmaf_rn(y, x, 2.0000714765e-1f);
    y = __fmaf_rn(y, x, -2.4999993993e-1f);
    y = __fmaf_rn(y, x, 3.3333331174e-1f);
    y = __fmul_rn(__fmul_rn(y, x), z);
    const float fe = (float)e;
    y = __fmaf_rn(fe, -2.12194440e-4f, y);
    y = __fmaf_rn(-0.5f, z, y);
    float r = __fadd_rn(x, y);
    r = __fmaf_rn(fe, 0.693359375f, r);
    return r;
}

__device__ __forceinline__ float cos2pi(float u) {
    const float t = __fmul_rn(u, 8.0f);
    const int j = (int)t;
    const float f = __fadd_rn(t, -(float)j);
    const float a = __fmul_rn((j & 1) ? __fadd_rn(1.0f, -f) : f, 0.78539816339744830962f);
    const float z = __fmul_rn(a, a);
    float s = -1.9515295891e-4f;
    s = __fmaf_rn(s, z, 8.3321608736e-3f);
    s = __fmaf_rn(s, z, -1.6666654611e-1f);
    s = __fmaf_rn(__fmul_rn(s, z), a, a);
    float c = 2.443315711809948e-5f;
    c = __fmaf_rn(c, z, -1.388731625493765e-3f);
    c = __fmaf_rn(c, z, 4.166664568298827e-2f);
    c = __fmaf_rn(c, __fmul_rn(z, z), __fmaf_rn(-0.5f, z, 1.0f));
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

__device__ __forceinline__ float normal01(float ua, float ub) {
    const float m = __fsqrt_rn(__fmul_rn(-2.0f, log01(ua)));
    return __fmul_rn(m, cos2pi(ub));
}

__device__ __forceinline__ float poisson(float lam, float ua, float ub) {
    if (!(lam > 0.0f)) return 0.0f;
    if (lam < 30.0f) {
        float p = exp_neg(lam), s = p;
        int n = 0;
        while (ua > s && n < 200) {
            ++n;
            p = __fdiv_rn(__fmul_rn(p, lam), (float)n);
            s = __fadd_rn(s, p);
        }
        return (float)n;
    }
    const float v = __fmaf_rn(__fsqrt_rn(lam), normal01(ua, ub), lam);
    const float n = rintf(v);
    return n > 0.0f ? n : 0.0f;
}

struct CcdArgs {
    long long n;
    float gain, sigma, adu_gain, full;
    int readout, photon, rnoise;
    unsigned k0, k1, frame;
};

__global__ void __launch_bounds__(256) k_ccd(const CcdArgs a, float *__restrict__ acc, const float *__restrict__ D,
                                             float *__restrict__ pixels) {
    // programmatic dependent launch: the CTAs are resident when the kernel that writes D drains
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < a.n; i += (long long)gridDim.x * blockDim.x) {
        float e = __fmaf_rn(a.gain, __ldg(&D[i]), acc[i]);
        if (!a.readout) { acc[i] = e; continue; }
        acc[i] = 0.0f;
        if (a.photon || a.rnoise) {
            unsigned w[4];
            philox4x32_10((unsigned)i, a.frame, 0u, 0u, a.k0, a.k1, w);
            if (a.photon) e = poisson(e, u01(w[0]), u01(w[1]));
            if (a.rnoise) e = __fmaf_rn(a.sigma, normal01(u01(w[2]), u01(w[3])), e);
        }
        if (a.adu_gain > 0.0f) {
            float v = rintf(__fdiv_rn(e, a.adu_gain));
            v = v > 0.0f ? v : 0.0f;
            e = v < a.full ? v : a.full;
        }
        pixels[i] = e;
    }
}

__global__ void __launch_bounds__(256) k_philox_test(unsigned k0, unsigned k1, unsigned frame, long long n, unsigned *__restrict__ out) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    unsigned w[4];
    philox4x32_10((unsigned)i, frame, 0u, 0u, k0, k1, w);
    reinterpret_cast<uint4 *>(out)[i] = make_uint4(w[0], w[1], w[2], w[3]);
}

// ================================================================ PupData from a reference frame
// One CTA: T = (Qa + Qb) + (Qc + Qd) per pixel, its maximum by a shared-memory tree (max is exact, so the order
// does not matter), then the flags.  Calibration-time, tiny.
__global__ void __launch_bounds__(1024) k_pupdata(int Nd, const float *__restrict__ ref, float thr, unsigned char *__restrict__ valid) {
    __shared__ float red[1024];
    const int Nq = Nd / 2, n = Nq * Nq;
    auto total = [&](int i) {
        const int Y = i / Nq, X = i % Nq;
        const float Qa = ref[(size_t)Y * Nd + X], Qb = ref[(size_t)Y * Nd + X + Nq];
        const float Qc = ref[(size_t)(Y + Nq) * Nd + X], Qd = ref[(size_t)(Y + Nq) * Nd + X + Nq];
        return __fadd_rn(__fadd_rn(Qa, Qb), __fadd_rn(Qc, Qd));
    };
    float m = 0.0f;
    for (int i = threadIdx.x; i < n; i += 1024) m = fmaxf(m, total(i));
    red[threadIdx.x] = m;
    __syncthreads();
    for (int w = 512; w > 0; w >>= 1) {
        if (threadIdx.x < w) red[threadIdx.x] = fmaxf(red[threadIdx.x], red[threadIdx.x + w]);
        __syncthreads();
    }
    const float cut = __fmul_rn(thr, red[0]);
    for (int i = threadIdx.x; i < n; i += 1024) valid[i] = total(i) >= cut ? 1 : 0;
}

// ================================================================ Modalrec
// modes[b][m] = sum_i R[m][i] sv[b][i].  Persistent grid, one CTA per SM; rows of R dealt round-robin.  R streams from
// HBM once, which bounds the kernel, so the job is to keep enough bytes in flight: thread 0 feeds a ring of NS row
// buffers in shared memory with one cp.async.bulk (1-D TMA copy, mbarrier completion) per row, NS rows ahead of the
// reduction -- 100 to 200 KB in flight per SM whatever the consumers are doing.  The CTA first gathers the compacted
// slope vectors of NB sources (index list built by the plan; its loads go out before griddepcontrol.wait, programmatic
// dependent launch) -- into registers when a row fits one sweep of the 256 threads (<= 8192 floats: thread t owns
// columns 4 t + 1024 k, so the shared-memory traffic is the row itself and nothing else), else through shared memory,
// one segment of a row per ring slot.  Four rows are reduced per iteration (4 NB independent sums per thread, one
// shuffle tree, one block barrier); per-lane partial sums, the eight warp sums and the segments of a row are added in
// a fixed order: deterministic.  Rows are padded to a multiple of 4 floats.
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s_stream(unsigned dst, const void *src, unsigned bytes, unsigned bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src),
                 "r"(bytes), "r"(bar)
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

constexpr int MR_THREADS = 512, MR_WARPS = MR_THREADS / 32;
constexpr int MR_SEG = 4 * 4 * MR_THREADS;        // most floats of a row per ring slot: four 16-byte loads per thread
constexpr int MR_EARLY = 4;                       // rows in flight before the gather (measured: 0: 28.6, 2: 28.6, 4: 26.8, 6: 28.4, 10: 30.4 us)
constexpr int MR_RP = 4;                          // chunks (rows, when a row fits a slot) reduced together

// NB: sources per walk over the rows; LPT: 16-byte loads per thread and chunk (ceil(seg / (4 MR_THREADS)), 1..4)
template <int NB, int LPT>
__global__ void __launch_bounds__(MR_THREADS, 1) k_modalrec(int n_modes, int ld, int B, int NS, int seg, size_t plane_stride,
                                                            const float *__restrict__ R, const int *__restrict__ idx,
                                                            const float *__restrict__ slopes, float *__restrict__ modes) {
    extern __shared__ __align__(16) float dsm[];  // ring [NS][seg] | sv [NB][ld] (when a row takes several segments)
    constexpr int RP = MR_RP, NW = MR_WARPS;
    __shared__ float part[2][RP][NB][NW];
    __shared__ __align__(8) unsigned long long bars[16];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nseg = (ld + seg - 1) / seg;        // seg: floats per ring slot (= ld when a row fits one slot)
    float *const sv = dsm + (size_t)NS * seg;
    const int rows_mine = n_modes > (int)blockIdx.x ? (n_modes - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;
    const int nchunks = rows_mine * nseg;         // chunk c = (row blockIdx.x + (c / nseg) gridDim.x, segment c % nseg)
    auto issue = [&](int c, int cbase) {          // thread 0; chunk c of this walk over the rows, the cbase + c-th the ring has seen
        const int m = blockIdx.x + (c / nseg) * gridDim.x, sg = c % nseg, slot = (cbase + c) % NS;
        const unsigned bytes = (unsigned)(min(seg, ld - sg * seg)) * 4u, bar = smem_u32(&bars[slot]);
        mbar_expect_tx(bar, bytes);
        bulk_g2s_stream(smem_u32(dsm + (size_t)slot * seg), R + (size_t)m * ld + (size_t)sg * seg, bytes, bar);
    };
    if (threadIdx.x == 0) {
        for (int i = 0; i < NS; ++i) mbar_init(smem_u32(&bars[i]), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    // The ring is primed in two steps: MR_EARLY rows before the gather (R does not depend on the step: the copies go out
    // before griddepcontrol.wait and keep the DRAM busy during the gather), the rest after the gather's loads have been
    // issued -- 148 x 200 KB of queued row copies ahead of them would make the gather wait for the whole first ring fill.
    const int early = min(NS, MR_EARLY);
    if (threadIdx.x == 0)
        for (int c = 0; c < early && c < nchunks; ++c) issue(c, 0);
    const int rp = NS < RP ? NS : RP;             // chunks per iteration (their slots are refilled after the iteration)
    for (int b0 = 0; b0 < B; b0 += NB) {
        const int nb = min(NB, B - b0);
        __syncthreads();                           // the barriers are initialised; (next batch) part has been read
        float4 svr[NB][LPT];
        if (nseg == 1) {
            int4 ic[LPT];                          // (idx is padded with -1 to the row length: all index loads, then all gathers)
#pragma unroll
            for (int k = 0; k < LPT; ++k) {
                const int c4 = (k * MR_THREADS + threadIdx.x) * 4;
                ic[k] = c4 < ld ? __ldg(reinterpret_cast<const int4 *>(idx + c4)) : make_int4(-1, -1, -1, -1);
            }
            asm volatile("griddepcontrol.wait;" ::: "memory");  // the slopes are complete (no-op after the first batch)
#pragma unroll
            for (int k = 0; k < LPT; ++k)
#pragma unroll
                for (int b = 0; b < NB; ++b) {
                    const float *__restrict__ sp = slopes + (size_t)(b0 + min(b, nb - 1)) * plane_stride;
                    svr[b][k].x = ic[k].x >= 0 && b < nb ? __ldg(&sp[ic[k].x]) : 0.0f;
                    svr[b][k].y = ic[k].y >= 0 && b < nb ? __ldg(&sp[ic[k].y]) : 0.0f;
                    svr[b][k].z = ic[k].z >= 0 && b < nb ? __ldg(&sp[ic[k].z]) : 0.0f;
                    svr[b][k].w = ic[k].w >= 0 && b < nb ? __ldg(&sp[ic[k].w]) : 0.0f;
                }
        } else {
            asm volatile("griddepcontrol.wait;" ::: "memory");
            for (int c = threadIdx.x; c < ld; c += blockDim.x) {
                const int ic = __ldg(&idx[c]);
#pragma unroll
                for (int b = 0; b < NB; ++b) sv[b * ld + c] = ic >= 0 && b < nb ? __ldg(&slopes[(size_t)(b0 + b) * plane_stride + ic]) : 0.0f;
            }
            __syncthreads();
        }
        // (a second batch of sources walks the rows again: chunk numbers keep counting, so slots and parities stay in step)
        const int cbase = (b0 / NB) * nchunks;
        if (threadIdx.x == 0)
            for (int c = b0 == 0 ? early : 0; c < NS && c < nchunks; ++c) issue(c, cbase);
        float racc = 0.0f;                         // (several segments per row) lane 0 of warp b: the sum over the segments so far
        int it = 0;
        for (int c0 = 0; c0 < nchunks; c0 += rp, ++it) {
            // rp chunks per iteration: rp NB independent sums per thread, one shuffle tree and ONE block barrier for all
            float acc[RP][NB];
#pragma unroll
            for (int r = 0; r < RP; ++r) {
#pragma unroll
                for (int b = 0; b < NB; ++b) acc[r][b] = 0.0f;
                const int c = c0 + r;
                if (r < rp && c < nchunks) {
                    const int cc = cbase + c, slot = cc % NS, sg = c % nseg, n4 = min(seg, ld - sg * seg) / 4;
                    mbar_wait(smem_u32(&bars[slot]), (cc / NS) & 1);
                    const float4 *__restrict__ row = reinterpret_cast<const float4 *>(dsm + (size_t)slot * seg);
                    float4 x[LPT];
#pragma unroll
                    for (int k = 0; k < LPT; ++k) {
                        const int c4 = k * MR_THREADS + threadIdx.x;
                        x[k] = c4 < n4 ? row[c4] : make_float4(0.f, 0.f, 0.f, 0.f);
                    }
#pragma unroll
                    for (int k = 0; k < LPT; ++k)
#pragma unroll
                        for (int b = 0; b < NB; ++b) {
                            const int c4 = min(k * MR_THREADS + (int)threadIdx.x, n4 - 1);
                            const float4 s_ = nseg == 1 ? svr[b][k] : *reinterpret_cast<const float4 *>(&sv[b * ld + sg * seg + 4 * c4]);
                            acc[r][b] = fmaf(x[k].x, s_.x, fmaf(x[k].y, s_.y, fmaf(x[k].z, s_.z, fmaf(x[k].w, s_.w, acc[r][b]))));
                        }
                }
            }
            const int buf = it & 1;
#pragma unroll
            for (int r = 0; r < RP; ++r)
#pragma unroll
                for (int b = 0; b < NB; ++b) {
                    float v = acc[r][b];
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
                    if (lane == 0) part[buf][r][b][warp] = v;
                }
            __syncthreads();                       // the slots have been read by every thread (part is double-buffered)
            if (threadIdx.x == 0)
                for (int r = 0; r < rp; ++r)
                    if (c0 + r + NS < nchunks) issue(c0 + r + NS, cbase);
            if (nseg == 1) {                       // warp (r, b): the NW warp sums of row r, source b, by a fixed tree
                const int r = warp / NB, b = warp % NB;
                if (r < rp && c0 + r < nchunks && b < nb) {
                    float v = lane < NW ? part[buf][r][b][lane] : 0.0f;
#pragma unroll
                    for (int o = NW / 2; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
                    if (lane == 0) modes[(size_t)(b0 + b) * n_modes + blockIdx.x + (c0 + r) * gridDim.x] = v;
                }
            } else if (warp < nb) {                // warp b: the chunks of the iteration in order, segments summed as they come
                for (int r = 0; r < rp && c0 + r < nchunks; ++r) {
                    const int c = c0 + r, sg = c % nseg;
                    float v = lane < NW ? part[buf][r][warp][lane] : 0.0f;
#pragma unroll
                    for (int o = NW / 2; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
                    racc = sg == 0 ? v : racc + v;
                    if (lane == 0 && sg == nseg - 1) modes[(size_t)(b0 + warp) * n_modes + blockIdx.x + (c / nseg) * gridDim.x] = racc;
                }
            }
        }
    }
}

typedef void (*modalrec_fn)(int, int, int, int, int, size_t, const float *, const int *, const float *, float *);
template <int NB>
modalrec_fn pick_modalrec_lpt(int lpt) {
    return lpt <= 1 ? k_modalrec<NB, 1> : lpt == 2 ? k_modalrec<NB, 2> : lpt == 3 ? k_modalrec<NB, 3> : k_modalrec<NB, 4>;
}
modalrec_fn pick_modalrec(int B, int lpt) {
    return B >= 4 ? pick_modalrec_lpt<4>(lpt) : B == 3 ? pick_modalrec_lpt<3>(lpt) : B == 2 ? pick_modalrec_lpt<2>(lpt) : pick_modalrec_lpt<1>(lpt);
}

}  // namespace

struct atmo_plan {
    AtmoArgs a;
    float *d_w;
    int device;
};

struct ccd_plan {
    long long n;
    int n_int, photon, rnoise, n_bits, device, grid;
    float sigma, adu_gain;
    unsigned long long seed;
    long long step;
    unsigned frame;
    float *d_acc;
};

struct modalrec_plan {
    int n_modes, Nq, nsv, ld, B, device, grid, NS, seg;
    size_t smem;
    float *d_R;
    int *d_idx;
    void (*fn)(int, int, int, int, int, size_t, const float *, const int *, const float *, float *);
};

extern "C" {

int chain_last_error(void) { return g_err; }
const char *chain_last_error_string(void) { return g_msg; }

// ---------------------------------------------------------------- atmosphere
atmo_plan *atmo_plan_create(int L, int S, int P, int B) {
    if (L < 1 || S < 2 || P < 1 || B < 1) { set_err(1, "atmo_plan_create: n_layers=%d, screen_side=%d, N_pup=%d, batch=%d", L, S, P, B); return nullptr; }
    if ((long long)L * B > ATMO_MAX || B > 65535 || P > 65535) { set_err(2, "atmo_plan_create: n_layers * batch = %d exceeds %d", L * B, ATMO_MAX); return nullptr; }
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { set_err(4, "no CUDA device: %s", cudaGetErrorString(cudaGetLastError())); return nullptr; }
    atmo_plan *p = new (std::nothrow) atmo_plan();
    if (!p) { set_err(3, "host allocation failed"); return nullptr; }
    p->device = dev;
    p->a.L = L; p->a.S = S; p->a.P = P; p->a.B = B;
    for (int l = 0; l < 16; ++l) p->a.w[l] = 1.0f;
    p->d_w = nullptr;
    if (cudaMalloc((void **)&p->d_w, sizeof(float) * (size_t)L) != cudaSuccess) {
        set_err(3, "atmo_plan_create: %s", cudaGetErrorString(cudaGetLastError()));
        delete p;
        return nullptr;
    }
    std::vector<float> ones((size_t)L, 1.0f);
    cudaMemcpy(p->d_w, ones.data(), sizeof(float) * (size_t)L, cudaMemcpyHostToDevice);
    return p;
}

int atmo_plan_set_weights(atmo_plan *p, const float *w) {
    if (!p) return set_err(1, "atmo_plan_set_weights: NULL plan");
    if (!on_device(p->device, "atmo_plan_set_weights")) return 1;
    std::vector<float> h((size_t)p->a.L, 1.0f);
    if (w) for (int l = 0; l < p->a.L; ++l) h[l] = w[l];
    for (int l = 0; l < p->a.L && l < 16; ++l) p->a.w[l] = h[l];
    if (cudaMemcpy(p->d_w, h.data(), sizeof(float) * h.size(), cudaMemcpyHostToDevice) != cudaSuccess)
        return set_err(4, "atmo_plan_set_weights: %s", cudaGetErrorString(cudaGetLastError()));
    return 0;
}

int atmo_propagate(atmo_plan *p, const float *screens, const double *shift, float *out, void *stream) {
    if (!p || !screens || !shift || !out) return set_err(1, "atmo_propagate: NULL argument");
    if (!on_device(p->device, "atmo_propagate")) return 1;
    AtmoArgs a = p->a;
    const int S = a.S;
    for (int i = 0; i < a.B * a.L; ++i) {
        const double dy = shift[2 * i], dx = shift[2 * i + 1];
        if (!std::isfinite(dy) || !std::isfinite(dx) || std::fabs(dy) > 1e15 || std::fabs(dx) > 1e15)
            return set_err(1, "atmo_propagate: shift %d is not finite", i);
        const double fy = std::floor(dy), fx = std::floor(dx);
        long long iy = (long long)std::fmod(fy, (double)S), ix = (long long)std::fmod(fx, (double)S);
        if (iy < 0) iy += S;
        if (ix < 0) ix += S;
        a.sh[i].iy = (int)iy; a.sh[i].ix = (int)ix;
        a.sh[i].fy = (float)(dy - fy); a.sh[i].fx = (float)(dx - fx);
        // (a fraction that rounds up to 1.0f in float32 is still right: weight 1 on the next sample)
    }
    a.vec = (a.P & 3) == 0 && (reinterpret_cast<uintptr_t>(out) & 15u) == 0;
    k_atmo<<<dim3((a.P + 511) / 512, a.P, a.B), 128, 0, (cudaStream_t)stream>>>(a, screens, p->d_w, out);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return set_err(4, "atmo_propagate: launch failed: %s", cudaGetErrorString(e));
    return 0;
}

void atmo_plan_destroy(atmo_plan *p) {
    if (!p) return;
    if (p->d_w) cudaFree(p->d_w);
    delete p;
}

// ---------------------------------------------------------------- CCD
ccd_plan *ccd_plan_create(long long n, int n_int, int photon, int rnoise, float sigma, float adu_gain, int n_bits,
                          unsigned long long seed) {
    if (n < 1 || n >= (1LL << 32) || n_int < 1 || !(sigma >= 0.0f) || !(adu_gain >= 0.0f) || n_bits < 1 || n_bits > 30 ||
        !std::isfinite(sigma) || !std::isfinite(adu_gain)) {
        set_err(1, "ccd_plan_create: n_pixels=%lld n_int=%d readout_level=%g adu_gain=%g n_bits=%d", n, n_int, (double)sigma, (double)adu_gain, n_bits);
        return nullptr;
    }
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { set_err(4, "no CUDA device: %s", cudaGetErrorString(cudaGetLastError())); return nullptr; }
    ccd_plan *p = new (std::nothrow) ccd_plan();
    if (!p) { set_err(3, "host allocation failed"); return nullptr; }
    p->n = n; p->n_int = n_int; p->photon = photon != 0; p->rnoise = rnoise != 0; p->n_bits = n_bits; p->device = dev;
    p->sigma = sigma; p->adu_gain = adu_gain; p->seed = seed; p->step = 0; p->frame = 0; p->d_acc = nullptr;
    const long long blocks = (n + 255) / 256, cap = (long long)sm_count() * 8;
    p->grid = (int)(blocks < cap ? blocks : cap);
    if (cudaMalloc((void **)&p->d_acc, sizeof(float) * (size_t)n) != cudaSuccess || cudaMemset(p->d_acc, 0, sizeof(float) * (size_t)n) != cudaSuccess) {
        set_err(3, "ccd_plan_create: %s", cudaGetErrorString(cudaGetLastError()));
        if (p->d_acc) cudaFree(p->d_acc);
        delete p;
        return nullptr;
    }
    return p;
}

int ccd_integrate(ccd_plan *p, const float *D, float gain, float *pixels, int *frame_ready, void *stream) {
    if (!p || !D) return set_err(1, "ccd_integrate: NULL plan or intensity");
    if (!on_device(p->device, "ccd_integrate")) return 1;
    const bool ready = (p->step + 1) % p->n_int == 0;
    if (ready && !pixels) return set_err(1, "ccd_integrate: this step reads a frame out and out_pixels is NULL");
    CcdArgs a;
    a.n = p->n; a.gain = gain; a.sigma = p->sigma; a.adu_gain = p->adu_gain; a.full = (float)((1u << p->n_bits) - 1u);
    a.readout = ready; a.photon = p->photon; a.rnoise = p->rnoise;
    a.k0 = (unsigned)p->seed; a.k1 = (unsigned)(p->seed >> 32); a.frame = p->frame;
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.gridDim = dim3(p->grid); cfg.blockDim = dim3(256); cfg.dynamicSmemBytes = 0; cfg.stream = (cudaStream_t)stream;
    cfg.attrs = at; cfg.numAttrs = 1;
    cudaLaunchKernelEx(&cfg, k_ccd, a, p->d_acc, D, pixels);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return set_err(4, "ccd_integrate: launch failed: %s", cudaGetErrorString(e));
    p->step += 1;
    if (ready) p->frame += 1;
    if (frame_ready) *frame_ready = ready ? 1 : 0;
    return 0;
}

int ccd_reset(ccd_plan *p, void *stream) {
    if (!p) return set_err(1, "ccd_reset: NULL plan");
    if (!on_device(p->device, "ccd_reset")) return 1;
    if (cudaMemsetAsync(p->d_acc, 0, sizeof(float) * (size_t)p->n, (cudaStream_t)stream) != cudaSuccess)
        return set_err(4, "ccd_reset: %s", cudaGetErrorString(cudaGetLastError()));
    p->step = 0; p->frame = 0;
    return 0;
}

void ccd_plan_destroy(ccd_plan *p) {
    if (!p) return;
    if (p->d_acc) cudaFree(p->d_acc);
    delete p;
}

int ccd_test_philox(unsigned long long seed, unsigned int frame, long long n, unsigned int *out, void *stream) {
    if (n < 1 || !out) return set_err(1, "ccd_test_philox: bad argument");
    k_philox_test<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>((unsigned)seed, (unsigned)(seed >> 32), frame, n, out);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return set_err(4, "ccd_test_philox: launch failed: %s", cudaGetErrorString(e));
    return 0;
}

// ---------------------------------------------------------------- PupData
int pupdata_from_frame(int Nd, const float *ref, float thr, unsigned char *host_valid, void *stream) {
    if (Nd < 2 || (Nd & 1) || !ref || !host_valid || !std::isfinite(thr)) return set_err(1, "pupdata_from_frame: bad argument");
    const size_t n = (size_t)(Nd / 2) * (Nd / 2);
    unsigned char *d = nullptr;
    if (cudaMalloc((void **)&d, n) != cudaSuccess) return set_err(3, "pupdata_from_frame: %s", cudaGetErrorString(cudaGetLastError()));
    k_pupdata<<<1, 1024, 0, (cudaStream_t)stream>>>(Nd, ref, thr, d);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaMemcpyAsync(host_valid, d, n, cudaMemcpyDeviceToHost, (cudaStream_t)stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize((cudaStream_t)stream);
    cudaFree(d);
    if (e != cudaSuccess) return set_err(4, "pupdata_from_frame: %s", cudaGetErrorString(e));
    return 0;
}

// ---------------------------------------------------------------- Modalrec
modalrec_plan *modalrec_plan_create(int n_modes, int Nq, const unsigned char *valid, const float *R, int B) {
    if (n_modes < 1 || Nq < 1 || B < 1 || !valid || !R) { set_err(1, "modalrec_plan_create: bad argument"); return nullptr; }
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { set_err(4, "no CUDA device: %s", cudaGetErrorString(cudaGetLastError())); return nullptr; }
    std::vector<int> idx;
    const int nq2 = Nq * Nq;
    for (int plane = 0; plane < 2; ++plane)
        for (int i = 0; i < nq2; ++i)
            if (valid[i]) idx.push_back(plane * nq2 + i);
    const int nsv = (int)idx.size();
    if (nsv < 1) { set_err(1, "modalrec_plan_create: no valid pixel"); return nullptr; }
    const int ld = (nsv + 3) & ~3;
    idx.resize((size_t)ld, -1);                    // (padded: the kernel reads whole int4s)
    // shared memory: the ring of row segments, and the slope vectors when a row takes more than one segment
    // (then in segments of 8192 floats, or shorter ones if the slope vectors leave no room for four of those);
    // nb sources share one walk over the rows of R: four if their slope vectors fit, else fewer (more walks)
    const size_t budget = 220 * 1024;
    int nb = B < 4 ? B : 4, seg = 0;
    size_t svb = 0, segb = 0;
    for (;; --nb) {
        svb = ld > MR_SEG ? (size_t)nb * ld * sizeof(float) : 0;
        seg = ld < MR_SEG ? ld : MR_SEG;
        while (seg > 1024 && svb + 4 * (size_t)seg * sizeof(float) > budget) seg /= 2;
        segb = (size_t)seg * sizeof(float);
        if (svb + 2 * segb <= budget || nb == 1) break;
    }
    if (svb + 2 * segb > budget) { set_err(2, "modalrec_plan_create: %d slopes do not fit shared memory (at most about 50 000)", nsv); return nullptr; }
    int NS = (int)((budget - svb) / segb);
    if (NS > 16) NS = 16;
    const size_t smem = svb + (size_t)NS * segb;
    modalrec_plan *p = new (std::nothrow) modalrec_plan();
    if (!p) { set_err(3, "host allocation failed"); return nullptr; }
    p->n_modes = n_modes; p->Nq = Nq; p->nsv = nsv; p->ld = ld; p->B = B; p->device = dev; p->smem = smem; p->NS = NS; p->seg = seg;
    p->d_R = nullptr; p->d_idx = nullptr;
    std::vector<float> Rp((size_t)n_modes * ld, 0.0f);
    for (int m = 0; m < n_modes; ++m) std::memcpy(&Rp[(size_t)m * ld], R + (size_t)m * nsv, sizeof(float) * (size_t)nsv);
    cudaError_t e = cudaMalloc((void **)&p->d_R, Rp.size() * sizeof(float));
    if (e == cudaSuccess) e = cudaMalloc((void **)&p->d_idx, idx.size() * sizeof(int));
    if (e == cudaSuccess) e = cudaMemcpy(p->d_R, Rp.data(), Rp.size() * sizeof(float), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(p->d_idx, idx.data(), idx.size() * sizeof(int), cudaMemcpyHostToDevice);
    p->fn = pick_modalrec(nb, (seg + 4 * MR_THREADS - 1) / (4 * MR_THREADS));
    const void *fn = (const void *)p->fn;
    if (e == cudaSuccess) e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) {
        set_err(e == cudaErrorMemoryAllocation ? 3 : 4, "modalrec_plan_create: %s", cudaGetErrorString(e));
        modalrec_plan_destroy(p);
        return nullptr;
    }
    // persistent: one CTA per SM (the gather of the slope vectors is paid once per CTA), rows dealt round-robin
    const int cap = sm_count();
    p->grid = n_modes < cap ? n_modes : cap;
    return p;
}

int modalrec_compute(modalrec_plan *p, const float *slopes, float *modes, void *stream) {
    if (!p || !slopes || !modes) return set_err(1, "modalrec_compute: NULL argument");
    if (!on_device(p->device, "modalrec_compute")) return 1;
    const size_t ps = (size_t)2 * p->Nq * p->Nq;
    cudaStream_t st = (cudaStream_t)stream;
    // programmatic dependent launch: the ring of rows of R is primed while the kernel before this one drains
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.gridDim = dim3(p->grid); cfg.blockDim = dim3(MR_THREADS); cfg.dynamicSmemBytes = p->smem; cfg.stream = st;
    cfg.attrs = at; cfg.numAttrs = 1;
    cudaLaunchKernelEx(&cfg, p->fn, p->n_modes, p->ld, p->B, p->NS, p->seg, ps, (const float *)p->d_R, (const int *)p->d_idx, slopes, modes);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return set_err(4, "modalrec_compute: launch failed: %s", cudaGetErrorString(e));
    return 0;
}

void modalrec_plan_destroy(modalrec_plan *p) {
    if (!p) return;
    if (p->d_R) cudaFree(p->d_R);
    if (p->d_idx) cudaFree(p->d_idx);
    delete p;
}

}  // extern "C"
