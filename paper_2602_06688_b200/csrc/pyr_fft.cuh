// pyr_fft.cuh -- in-register radix-4/8/16 butterflies and the per-line operator
//
//     out = IDFT_N( g . DFT_N( zero-padded in ) )          (un-normalised)
//
// used by both passes of the separable pyramid propagation.
// A line of N complex64 samples is owned by a group of TPL = N/16 threads, 16 samples per
// thread.  N = N1*N2*N3; the forward transform is decimation-in-frequency (natural order in,
// digit-reversed out), the mask multiply happens in digit-reversed order on the registers
// that the last forward butterfly produced, and the inverse transform is the exact mirror
// (decimation-in-time, digit-reversed in, natural out), so no reordering pass exists and the
// mask multiply sits between the last forward and the first inverse butterfly of the same
// thread (north_star item 4).  Between passes the group exchanges data through a private
// shared-memory line; every exchange is "in place" (a thread writes exactly the slots it
// read), which leaves one group barrier per exchange.
//
// What keeps the LSU pipe free for those exchanges (profiles/README.md, r1a -> r1b):
//   * every twiddle a thread ever needs depends only on its lane position, so it is loaded
//     ONCE into registers (struct Twid) and reused for all modulation points of the line;
//   * the built-in pyramid mask costs no instruction: in the half-band form (pyr.cu) it is a
//     real sign pattern that folds into the first inverse butterfly and the last inverse load;
//   * shared-memory slots are a per-thread base plus a compile-time offset;
//   * the first forward butterfly is pruned: only the first N1/PRUNE inputs can be non-zero
//     (the pupil occupies P <= N/PRUNE samples of the padded line).
#pragma once
#include <cuda_runtime.h>

#include <utility>

namespace pyr {

// ---------------------------------------------------------------- complex helpers
// A complex64 sample is a float2 in an aligned register pair.  sm_100a has packed FP32x2
// instructions (FADD2 / FMUL2 / FFMA2; PTX add/mul/fma.rn.f32x2) that run on the same 128
// FP32 lanes per SM as the scalar ones -- same flops per clock (measured: 127 lane-ops per SM
// per clock either way) -- but take ONE issue slot for two lanes.  The line operator is bound
// by instruction issue (profiles/README.md, r1c), so every complex add is one FADD2 and every
// complex multiply one FMUL2 + one FFMA2; ptxas folds the lo/hi swaps, the per-half negations
// and the scalar broadcasts written below into operand modifiers (.LO_HI, .NP, .F32), so
// multiplying by +-i costs nothing.
typedef unsigned long long u64;
__device__ __forceinline__ u64 pk(float2 a) {
    u64 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a.x), "f"(a.y));
    return r;
}
__device__ __forceinline__ float2 upk(u64 r) {
    float2 a;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(a.x), "=f"(a.y) : "l"(r));
    return a;
}
__device__ __forceinline__ float2 add2(float2 a, float2 b) {
    u64 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk(a)), "l"(pk(b)));
    return upk(r);
}
__device__ __forceinline__ float2 sub2(float2 a, float2 b) {
    u64 r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk(a)), "l"(pk(b)));
    return upk(r);
}
__device__ __forceinline__ float2 mul2(float2 a, float2 b) {
    u64 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk(a)), "l"(pk(b)));
    return upk(r);
}
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) {
    u64 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(pk(a)), "l"(pk(b)), "l"(pk(c)));
    return upk(r);
}
__device__ __forceinline__ float2 bc(float s) { return make_float2(s, s); }
__device__ __forceinline__ float2 swp(float2 a) { return make_float2(a.y, a.x); }

__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return add2(a, b); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return sub2(a, b); }
// a * b = b.x * (a.x, a.y) + b.y * (-a.y, a.x)
__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
    const float2 t = mul2(bc(b.y), swp(a));
    return fma2(bc(b.x), a, make_float2(-t.x, t.y));
}
// a * conj(b) = b.x * (a.x, a.y) + b.y * (a.y, -a.x)
__device__ __forceinline__ float2 cmulc(float2 a, float2 b) {
    const float2 t = mul2(bc(b.y), swp(a));
    return fma2(bc(b.x), a, make_float2(t.x, -t.y));
}
// Twiddle tables hold the FORWARD factors exp(-2 pi i ...); the inverse uses their conjugates.
template <int SIGN>
__device__ __forceinline__ float2 twmul(float2 a, float2 w) { return SIGN < 0 ? cmul(a, w) : cmulc(a, w); }
// multiply by SIGN * i
template <int SIGN>
__device__ __forceinline__ float2 roti(float2 a) {
    return SIGN < 0 ? make_float2(a.y, -a.x) : make_float2(-a.y, a.x);
}
// multiply by the compile-time constant (cr + i * SIGN * ci)
template <int SIGN>
__device__ __forceinline__ float2 cmulk(float2 a, float cr, float ci) {
    const float s = SIGN < 0 ? -ci : ci;
    const float2 t = mul2(bc(s), swp(a));
    return fma2(bc(cr), a, make_float2(-t.x, t.y));
}

#define PYR_SQRT1_2 0.70710678118654752440f
#define PYR_COS_PI_8 0.92387953251128675613f
#define PYR_SIN_PI_8 0.38268343236508977173f

// multiply by exp(SIGN * 2 pi i q / 16); q is a constant after unrolling, so the switch folds.
template <int SIGN>
__device__ __forceinline__ float2 mul_root16(float2 a, int q) {
    switch (q & 15) {
        case 0:  return a;
        case 1:  return cmulk<SIGN>(a, PYR_COS_PI_8, PYR_SIN_PI_8);
        case 2:  return cmulk<SIGN>(a, PYR_SQRT1_2, PYR_SQRT1_2);
        case 3:  return cmulk<SIGN>(a, PYR_SIN_PI_8, PYR_COS_PI_8);
        case 4:  return roti<SIGN>(a);
        case 5:  return cmulk<SIGN>(a, -PYR_SIN_PI_8, PYR_COS_PI_8);
        case 6:  return cmulk<SIGN>(a, -PYR_SQRT1_2, PYR_SQRT1_2);
        case 7:  return cmulk<SIGN>(a, -PYR_COS_PI_8, PYR_SIN_PI_8);
        case 8:  return make_float2(-a.x, -a.y);
        case 9:  return cmulk<SIGN>(a, -PYR_COS_PI_8, -PYR_SIN_PI_8);
        case 10: return cmulk<SIGN>(a, -PYR_SQRT1_2, -PYR_SQRT1_2);
        case 11: return cmulk<SIGN>(a, -PYR_SIN_PI_8, -PYR_COS_PI_8);
        case 12: return roti<-SIGN>(a);
        case 13: return cmulk<SIGN>(a, PYR_SIN_PI_8, -PYR_COS_PI_8);
        case 14: return cmulk<SIGN>(a, PYR_SQRT1_2, -PYR_SQRT1_2);
        default: return cmulk<SIGN>(a, PYR_COS_PI_8, -PYR_SIN_PI_8);
    }
}

// ---------------------------------------------------------------- butterflies (natural order in and out)
// X[k] = sum_n x[n] exp(SIGN * 2 pi i n k / R)
template <int SIGN>
__device__ __forceinline__ void dft2(float2 &a, float2 &b) {
    float2 t = a;
    a = cadd(t, b);
    b = csub(t, b);
}

template <int SIGN>
__device__ __forceinline__ void dft4(float2 &a0, float2 &a1, float2 &a2, float2 &a3) {
    float2 t0 = cadd(a0, a2), t1 = csub(a0, a2);
    float2 t2 = cadd(a1, a3), t3 = roti<SIGN>(csub(a1, a3));
    a0 = cadd(t0, t2);
    a2 = csub(t0, t2);
    a1 = cadd(t1, t3);
    a3 = csub(t1, t3);
}

// dft4 of (a0, a1, -a2, -a3): the negation swaps the roles of the first layer's sums and differences.
template <int SIGN>
__device__ __forceinline__ void dft4n(float2 &a0, float2 &a1, float2 &a2, float2 &a3) {
    float2 t0 = csub(a0, a2), t1 = cadd(a0, a2);
    float2 t2 = csub(a1, a3), t3 = roti<SIGN>(cadd(a1, a3));
    a0 = cadd(t0, t2);
    a2 = csub(t0, t2);
    a1 = cadd(t1, t3);
    a3 = csub(t1, t3);
}

// NEG: the inputs v[4..8) are taken negated (upper half of the band, see LineConv HALF mask).
template <int SIGN, bool NEG = false>
__device__ __forceinline__ void dft8(float2 *v) {
    // n = n0 + 2 n1, k = k1 + 4 k0
    if (NEG) {
        dft4n<SIGN>(v[0], v[2], v[4], v[6]);
        dft4n<SIGN>(v[1], v[3], v[5], v[7]);
    } else {
        dft4<SIGN>(v[0], v[2], v[4], v[6]);   // y[0][k1] -> v[2 k1]
        dft4<SIGN>(v[1], v[3], v[5], v[7]);   // y[1][k1] -> v[2 k1 + 1]
    }
    v[3] = mul2(bc(PYR_SQRT1_2), cadd(v[3], roti<SIGN>(v[3])));    // W8^1 = (1 + SIGN i)/sqrt2
    v[5] = roti<SIGN>(v[5]);                                       // W8^2 = SIGN i
    v[7] = mul2(bc(PYR_SQRT1_2), csub(roti<SIGN>(v[7]), v[7]));    // W8^3 = (-1 + SIGN i)/sqrt2
    float2 x0 = cadd(v[0], v[1]), x4 = csub(v[0], v[1]);
    float2 x1 = cadd(v[2], v[3]), x5 = csub(v[2], v[3]);
    float2 x2 = cadd(v[4], v[5]), x6 = csub(v[4], v[5]);
    float2 x3 = cadd(v[6], v[7]), x7 = csub(v[6], v[7]);
    v[0] = x0; v[1] = x1; v[2] = x2; v[3] = x3; v[4] = x4; v[5] = x5; v[6] = x6; v[7] = x7;
}

// NEG: the inputs v[8..16) are taken negated.
template <int SIGN, bool NEG = false>
__device__ __forceinline__ void dft16(float2 *v) {
    // n = n0 + 4 n1, k = k1 + 4 k0
#pragma unroll
    for (int n0 = 0; n0 < 4; ++n0) {   // y[n0][k1] -> v[n0 + 4 k1]
        if (NEG) dft4n<SIGN>(v[n0], v[n0 + 4], v[n0 + 8], v[n0 + 12]);
        else dft4<SIGN>(v[n0], v[n0 + 4], v[n0 + 8], v[n0 + 12]);
    }
    // twiddles W16^(n0 k1)
    v[5] = cmulk<SIGN>(v[5], PYR_COS_PI_8, PYR_SIN_PI_8);      // n0=1,k1=1 : W^1
    v[9] = cmulk<SIGN>(v[9], PYR_SQRT1_2, PYR_SQRT1_2);        // n0=1,k1=2 : W^2
    v[13] = cmulk<SIGN>(v[13], PYR_SIN_PI_8, PYR_COS_PI_8);    // n0=1,k1=3 : W^3
    v[6] = cmulk<SIGN>(v[6], PYR_SQRT1_2, PYR_SQRT1_2);        // n0=2,k1=1 : W^2
    v[10] = roti<SIGN>(v[10]);                                 // n0=2,k1=2 : W^4
    v[14] = cmulk<SIGN>(v[14], -PYR_SQRT1_2, PYR_SQRT1_2);     // n0=2,k1=3 : W^6
    v[7] = cmulk<SIGN>(v[7], PYR_SIN_PI_8, PYR_COS_PI_8);      // n0=3,k1=1 : W^3
    v[11] = cmulk<SIGN>(v[11], -PYR_SQRT1_2, PYR_SQRT1_2);     // n0=3,k1=2 : W^6
    v[15] = cmulk<SIGN>(v[15], -PYR_COS_PI_8, -PYR_SIN_PI_8);  // n0=3,k1=3 : W^9
#pragma unroll
    for (int k1 = 0; k1 < 4; ++k1) dft4<SIGN>(v[4 * k1], v[4 * k1 + 1], v[4 * k1 + 2], v[4 * k1 + 3]);  // X[k1 + 4 k0] -> v[4 k1 + k0]
    float2 o[16];
#pragma unroll
    for (int k1 = 0; k1 < 4; ++k1)
#pragma unroll
        for (int k0 = 0; k0 < 4; ++k0) o[k1 + 4 * k0] = v[4 * k1 + k0];
#pragma unroll
    for (int k = 0; k < 16; ++k) v[k] = o[k];
}

// 32-point DFT as five radix-2 decimation-in-time layers with the twiddle of each butterfly in tangent form:
// a +- w b with w = c (1 + i t) is u = b + t (i b), a +- c u -- three packed FMAs where multiply-then-add takes
// four (|t| <= 1: for |sin| > |cos| the factor is written i s (1 - i t) instead).  80 butterflies, 34 of them
// with a twiddle other than 1 or +-i: 194 packed instructions (a 4 x 8 split with separate twiddle multiplies: 216).
// FFMA2 cannot negate ONE half of a multiplicand, so the per-half signs sit in constant pairs (-t, t), (-S, S): six
// register pairs per kernel.  Natural order in and out.
// NZA: only inputs x[n], n < 8 NZA, can be non-zero (pruned first forward butterfly; v[8 NZA .. 32) is ignored on
// entry): the first one or two layers are copies.  NEG: the inputs v[16..32) are taken negated (swaps the sums and
// differences of the first layer).
__host__ __device__ constexpr float cos32(int q) {   // cos(2 pi q / 32), 0 <= q <= 16
    return q == 0 ? 1.0f : q == 1 ? 0.98078528040323044913f : q == 2 ? 0.92387953251128675613f : q == 3 ? 0.83146961230254523708f
         : q == 4 ? 0.70710678118654752440f : q == 5 ? 0.55557023301960222474f : q == 6 ? 0.38268343236508977173f
         : q == 7 ? 0.19509032201612826785f : q == 8 ? 0.0f : -cos32(16 - q);
}
__host__ __device__ constexpr float sin32(int q) { return q <= 8 ? cos32(8 - q) : cos32(q - 8); }   // sin(2 pi q / 32), 0 <= q <= 16

// (a, b) <- (a + w b, a - w b), w = exp(SIGN 2 pi i Q / 32), 0 <= Q < 16
template <int SIGN, int Q>
__device__ __forceinline__ void bfly32(float2 &a, float2 &b) {
    const float2 a0 = a;
    if constexpr (Q == 0) {
        a = cadd(a0, b);
        b = csub(a0, b);
    } else if constexpr (Q == 8) {
        const float2 r = roti<SIGN>(b);
        a = cadd(a0, r);
        b = csub(a0, r);
    } else if constexpr (Q == 4 || Q == 12) {  // w = c (1 +- SIGN i): u by one packed add (per-half negation folds into FADD2)
        constexpr float c = cos32(Q);
        const float2 u = Q == 4 ? cadd(b, roti<SIGN>(b)) : csub(b, roti<SIGN>(b));
        a = fma2(bc(c), u, a0);
        b = fma2(bc(-c), u, a0);
    } else if constexpr (Q < 4 || Q > 12) {    // |cos| > |sin|: w = c (1 + i t), t = SIGN sin / cos
        constexpr float c = cos32(Q), t = (SIGN < 0 ? -sin32(Q) : sin32(Q)) / cos32(Q);
        const float2 u = fma2(make_float2(-t, t), swp(b), b);
        a = fma2(bc(c), u, a0);
        b = fma2(bc(-c), u, a0);
    } else {                                   // w = i S (1 - i t), S = SIGN sin, t = cos / S;  w b = S (i u), u = b - t (i b)
        constexpr float S = SIGN < 0 ? -sin32(Q) : sin32(Q), t = cos32(Q) / S;
        const float2 u = fma2(make_float2(t, -t), swp(b), b), su = swp(u);
        a = fma2(make_float2(-S, S), su, a0);
        b = fma2(make_float2(S, -S), su, a0);
    }
}
// one radix-2 layer of span M over the 32 values: butterfly I pairs o[k0 + j], o[k0 + j + M/2] with twiddle W32^(j 32/M)
template <int SIGN, int M, int... I>
__device__ __forceinline__ void layer32(float2 *o, std::integer_sequence<int, I...>) {
    (bfly32<SIGN, (I % (M / 2)) * (32 / M)>(o[(I / (M / 2)) * M + I % (M / 2)], o[(I / (M / 2)) * M + I % (M / 2) + M / 2]), ...);
}

template <int SIGN, int NZA = 4, bool NEG = false>
__device__ __forceinline__ void dft32(float2 *v) {
    static_assert(!(NEG && NZA != 4), "negated half needs all inputs");
    float2 o[32];
    // bit-reversed input order: o[i] = x[rev5(i)]; layer 1 pairs x[n], x[n + 16], layer 2 adds x[n + 8], x[n + 24]
#pragma unroll
    for (int i = 0; i < 32; ++i) {
        const int r = ((i & 1) << 4) | ((i & 2) << 2) | (i & 4) | ((i & 8) >> 2) | ((i & 16) >> 4);
        o[i] = v[r];
    }
    // layer 1 (M = 2): o[2p], o[2p + 1] = x[n], x[n + 16]
#pragma unroll
    for (int p = 0; p < 16; ++p) {
        if (NZA == 4) {
            const float2 a = o[2 * p], b = o[2 * p + 1];
            o[2 * p] = NEG ? csub(a, b) : cadd(a, b);
            o[2 * p + 1] = NEG ? cadd(a, b) : csub(a, b);
        } else {
            o[2 * p + 1] = o[2 * p];               // x[n + 16] = 0
        }
    }
    // layer 2 (M = 4): groups (x[n], x[n + 16] | x[n + 8], x[n + 24]); NZA == 1: the second pair is zero
    if (NZA == 1) {
#pragma unroll
        for (int k0 = 0; k0 < 32; k0 += 4) {
            o[k0 + 2] = o[k0];
            o[k0 + 3] = o[k0 + 1];
        }
    } else {
        layer32<SIGN, 4>(o, std::make_integer_sequence<int, 16>{});
    }
    layer32<SIGN, 8>(o, std::make_integer_sequence<int, 16>{});
    layer32<SIGN, 16>(o, std::make_integer_sequence<int, 16>{});
    layer32<SIGN, 32>(o, std::make_integer_sequence<int, 16>{});
#pragma unroll
    for (int k = 0; k < 32; ++k) v[k] = o[k];
}

template <int R, int SIGN>
__device__ __forceinline__ void dftR(float2 *v) {
    if (R == 32) dft32<SIGN>(v);
    else if (R == 16) dft16<SIGN>(v);
    else if (R == 8) dft8<SIGN>(v);
    else if (R == 4) dft4<SIGN>(v[0], v[1], v[2], v[3]);
    else if (R == 2) dft2<SIGN>(v[0], v[1]);
}
// R-point DFT of (v[0..R/2), -v[R/2..R)), R >= 4
template <int R, int SIGN>
__device__ __forceinline__ void dftR_neg(float2 *v) {
    static_assert(R >= 4, "negated-half butterfly needs R >= 4");
    if (R == 32) dft32<SIGN, 4, true>(v);
    else if (R == 16) dft16<SIGN, true>(v);
    else if (R == 8) dft8<SIGN, true>(v);
    else dft4n<SIGN>(v[0], v[1], v[2], v[3]);
}
// Forward R-point DFT of which only inputs 0..NZ-1 can be non-zero (v[NZ..R) is ignored on
// entry).  With R = NZ*Q and k = b + Q a:  X[b + Q a] = DFT_NZ( x[n] W_R^(n b) )[a].
template <int R, int NZ>
__device__ __forceinline__ void dft_pruned_fwd(float2 *v) {
    if (NZ >= R) {
        dftR<R, -1>(v);
    } else if (R == 32) {
        dft32<-1, (NZ >= 8 ? NZ / 8 : 1)>(v);
    } else {
        constexpr int Q = R / NZ;
        float2 y[Q][NZ];
#pragma unroll
        for (int b = 0; b < Q; ++b) {
#pragma unroll
            for (int n = 0; n < NZ; ++n) y[b][n] = mul_root16<-1>(v[n], n * b * (16 / R));
            dftR<NZ, -1>(y[b]);
        }
#pragma unroll
        for (int b = 0; b < Q; ++b)
#pragma unroll
            for (int a = 0; a < NZ; ++a) v[b + Q * a] = y[b][a];
    }
}

// ---------------------------------------------------------------- factorisations
// Chosen so that, with the padding of Line::pad, all three exchange patterns are free of
// shared-memory bank conflicts (512 = 8*8*8 and 1024 = 16*8*8 are not: 2-way on pattern B).
template <int N, int E = 16> struct Fac;
template <> struct Fac<16, 16>   { static constexpr int N1 = 16, N2 = 1,  N3 = 1; };
template <> struct Fac<32, 16>   { static constexpr int N1 = 8,  N2 = 4,  N3 = 1; };
template <> struct Fac<64, 16>   { static constexpr int N1 = 8,  N2 = 8,  N3 = 1; };
template <> struct Fac<128, 16>  { static constexpr int N1 = 16, N2 = 8,  N3 = 1; };
template <> struct Fac<256, 16>  { static constexpr int N1 = 16, N2 = 16, N3 = 1; };
template <> struct Fac<512, 16>  { static constexpr int N1 = 4,  N2 = 16, N3 = 8; };
template <> struct Fac<1024, 16> { static constexpr int N1 = 8,  N2 = 8,  N3 = 16; };
template <> struct Fac<2048, 16> { static constexpr int N1 = 16, N2 = 16, N3 = 8; };
// 32 samples per thread: one warp owns a 1024-point line, two passes, one exchange per transform
template <> struct Fac<1024, 32> { static constexpr int N1 = 32, N2 = 32, N3 = 1; };

// ---------------------------------------------------------------- line geometry
template <int N, int E = 16>
struct Line {
    static constexpr int N1 = Fac<N, E>::N1, N2 = Fac<N, E>::N2, N3 = Fac<N, E>::N3;
    static constexpr int EPT = E;              // samples per thread
    static constexpr int TPL = N / EPT;        // threads per line
    static constexpr int S1 = N / N1;          // = N2*N3, stride of the first-pass butterfly
    static constexpr int RL = N3 > 1 ? N3 : (N2 > 1 ? N2 : N1);   // radix of the last forward pass
    static constexpr int B1 = E / N1, B2 = E / N2, B3 = E / N3, BL = E / RL;   // butterflies per thread
    // shared-memory slot of logical position p (float2 units); padding keeps the strided
    // accesses of the exchanges off the same banks.
    static constexpr int PS = E == 32 ? 5 : 4;
    __host__ __device__ static constexpr int pad(int p) { return p + (p >> PS); }
    static constexpr int SMEM_LINE = ((N + (N >> PS) + 1) + 1) & ~1;   // float2 per line, even
    static_assert(N1 * N2 * N3 == N, "factorisation");
};

// group barrier: the TPL threads that own one line.
template <int TPL>
__device__ __forceinline__ void group_sync(int group) {
    if (TPL <= 32) {
        __syncwarp();
    } else {
        asm volatile("bar.sync %0, %1;" ::"r"(group + 1), "r"(TPL) : "memory");
    }
}

// ---------------------------------------------------------------- per-thread constants of a line
//   tw1[k1*S1 + m]  = exp(-2 pi i m k1 / N)           (table, N entries)
//   tw2[k2*N3 + n3] = exp(-2 pi i n3 k2 / (N2*N3))    (table, N2*N3 entries)
// A thread's twiddles depend only on its position t in the group, so they are read once.
// Shared-memory slots are pad(base) + compile-time offset (the three access patterns of the
// exchanges separate; checked exhaustively on the host for every supported N):
//   A  slot(k1*S1 + m)           = a[i] + k1*(S1 + S1/16)            (S1 % 16 == 0, else pad() in full)
//   B  slot(k1*S1 + n2*N3 + n3)  = b[i] + n2*N3 + ((n2*N3) >> 4)
//   C  slot(c*N3 + n3)           = c[i] + n3
template <int N, int E = 16>
struct Twid {
    using L = Line<N, E>;
    static constexpr bool SEP_A = (L::S1 % (1 << L::PS) == 0);
    float2 w1[L::B1][L::N1];    // [i][k1], k1 = 0 unused
    // w2 depends on the thread through n3 = (t + TPL*i) % N3 only: one copy when N3 | TPL
    static constexpr bool W2_ONE = (L::TPL % L::N3 == 0);
    float2 w2[W2_ONE ? 1 : L::B2][L::N2];    // [i][k2], k2 = 0 unused (only when N3 > 1)
    __device__ __forceinline__ const float2 &w2at(int i, int k2) const { return w2[W2_ONE ? 0 : i][k2]; }
    int a[L::B1], b[L::B2], c[L::B3];

    __device__ __forceinline__ void load(int t, const float2 *__restrict__ tw1, const float2 *__restrict__ tw2) {
        if (L::N2 > 1) {
#pragma unroll
            for (int i = 0; i < L::B1; ++i) {
                const int m = t + L::TPL * i;
                a[i] = SEP_A ? L::pad(m) : m;
#pragma unroll
                for (int k1 = 1; k1 < L::N1; ++k1) w1[i][k1] = __ldg(&tw1[k1 * L::S1 + m]);
            }
#pragma unroll
            for (int i = 0; i < L::B2; ++i) {
                const int cc = t + L::TPL * i, k1 = cc / L::N3, n3 = cc % L::N3;
                b[i] = L::pad(k1 * L::S1 + n3);
            }
        }
        if (L::N3 > 1) {
#pragma unroll
            for (int i = 0; i < (W2_ONE ? 1 : L::B2); ++i) {
                const int n3 = (t + L::TPL * i) % L::N3;
#pragma unroll
                for (int k2 = 1; k2 < L::N2; ++k2) w2[i][k2] = __ldg(&tw2[k2 * L::N3 + n3]);
            }
#pragma unroll
            for (int i = 0; i < L::B3; ++i) c[i] = L::pad((t + L::TPL * i) * L::N3);
        }
    }
    __device__ __forceinline__ int slotA(int i, int k1) const {
        return SEP_A ? a[i] + k1 * (L::S1 + (L::S1 >> L::PS)) : L::pad(k1 * L::S1 + a[i]);
    }
    __device__ __forceinline__ int slotB(int i, int n2) const { return b[i] + n2 * L::N3 + ((n2 * L::N3) >> L::PS); }
    __device__ __forceinline__ int slotC(int i, int n3) const { return c[i] + n3; }
};

// ---------------------------------------------------------------- the line operator
// Register layout on entry  : v[i*N1 + n1] = x[n1*S1 + m_i],  m_i = t + TPL*i,  i < 16/N1; only
//                             n1 < N1/PRUNE is read (the rest of the padded line is zero).
// Register layout on return : the same, all n1, holding IDFT(g . DFT(x)) (un-normalised).
// Layout at the mask multiply: v[i*RL + q] is position p = (t + TPL*i)*RL + q of the
// digit-reversed spectrum, p = (k1*N2 + k2)*N3 + k3  <->  frequency k1 + N1*k2 + N1*N2*k3.
// HALF = false : `gperm`, any 1-D mask as a global table: the value for position p = (t + TPL*i)*RL + q
//                sits at (i*RL + q)*TPL + t, so that a warp reads consecutive entries.
// HALF = true  : the real sign mask m(u) = (-1)^u * (u < N/2 ? 1 : -1) of the half-length form of
//                the pyramid operator (pyr.cu, "half-band split").  N1 is even, so (-1)^u =
//                (-1)^k1: it commutes with the inverse passes over k3 and k2 and is applied as a
//                compile-time negation where k1 becomes a register index (the load of the last
//                inverse pass); "u >= N/2" is the upper half of the last forward butterfly's
//                outputs, i.e. the first inverse butterfly takes its upper inputs negated, which
//                only swaps sums and differences of its first layer.  No instruction, exact.
//
// The operator is cut into segments separated by the shared-memory exchanges:
//   s0 : pruned first forward butterfly, twiddle w1                      -> store A
//   s1 : load B, radix N2, twiddle w2                                    -> store B   (N3 > 1)
//   s2 : load C (B if N3 == 1), last forward butterfly, mask, first inverse butterfly -> store C (B)
//   s3 : load B, conj w2, radix N2                                       -> store B   (N3 > 1)
//   s4 : load A, conj w1, mask rotation, radix N1
// run() executes them for one line with a group barrier per exchange.
template <int N, int PRUNE, bool HALF, int E = 16>
struct LineConv {
    using L = Line<N, E>;
    static constexpr int N1 = L::N1, N2 = L::N2, N3 = L::N3, TPL = L::TPL, S1 = L::S1, RL = L::RL;
    static constexpr int NZ = N1 / PRUNE;     // non-zero inputs of a first-pass butterfly
    using TW = Twid<N, E>;

    // ---- s0
    __device__ static __forceinline__ void s0_a(float2 *v) {
#pragma unroll
        for (int i = 0; i < L::B1; ++i) dft_pruned_fwd<N1, NZ>(v + i * N1);
    }
    __device__ static __forceinline__ void s0_b(float2 *v, float2 *sm, const TW &tw) {
#pragma unroll
        for (int i = 0; i < L::B1; ++i)
#pragma unroll
            for (int k1 = 0; k1 < N1; ++k1) {
                float2 a = v[i * N1 + k1];
                if (k1 > 0) a = cmul(a, tw.w1[i][k1]);
                sm[tw.slotA(i, k1)] = a;
            }
    }
    // ---- s1 (N3 > 1)
    __device__ static __forceinline__ void s1_ld(float2 *v, const float2 *sm, const TW &tw) {
#pragma unroll
        for (int i = 0; i < L::B2; ++i)
#pragma unroll
            for (int n2 = 0; n2 < N2; ++n2) v[i * N2 + n2] = sm[tw.slotB(i, n2)];
    }
    __device__ static __forceinline__ void s1_a(float2 *v) {
#pragma unroll
        for (int i = 0; i < L::B2; ++i) dftR<N2, -1>(v + i * N2);
    }
    __device__ static __forceinline__ void s1_b(float2 *v, float2 *sm, const TW &tw) {
#pragma unroll
        for (int i = 0; i < L::B2; ++i)
#pragma unroll
            for (int k2 = 0; k2 < N2; ++k2) {
                float2 a = v[i * N2 + k2];
                if (k2 > 0) a = cmul(a, tw.w2at(i, k2));
                sm[tw.slotB(i, k2)] = a;
            }
    }
    // ---- s2
    __device__ static __forceinline__ void s2_ld(float2 *v, const float2 *sm, const TW &tw) {
        if (N3 > 1) {
#pragma unroll
            for (int i = 0; i < L::B3; ++i)
#pragma unroll
                for (int n3 = 0; n3 < N3; ++n3) v[i * N3 + n3] = sm[tw.slotC(i, n3)];
        } else {
            s1_ld(v, sm, tw);
        }
    }
    __device__ static __forceinline__ void s2_a(float2 *v) {   // last forward butterfly
#pragma unroll
        for (int i = 0; i < L::BL; ++i) dftR<RL, -1>(v + i * RL);
    }
    __device__ static __forceinline__ void s2_b(float2 *v, int t, const TW &tw, const float2 *__restrict__ gperm) {
        if (HALF) {
#pragma unroll
            for (int i = 0; i < L::BL; ++i) dftR_neg<RL, +1>(v + i * RL);
        } else {
#pragma unroll
            for (int i = 0; i < L::BL; ++i) {
#pragma unroll
                for (int q = 0; q < RL; ++q) v[i * RL + q] = cmul(v[i * RL + q], __ldg(&gperm[(i * RL + q) * TPL + t]));
                dftR<RL, +1>(v + i * RL);
            }
        }
    }
    __device__ static __forceinline__ void s2_st(const float2 *v, float2 *sm, const TW &tw) {
        if (N3 > 1) {
#pragma unroll
            for (int i = 0; i < L::B3; ++i)
#pragma unroll
                for (int n3 = 0; n3 < N3; ++n3) sm[tw.slotC(i, n3)] = v[i * N3 + n3];
        } else {
            s3_st(v, sm, tw);
        }
    }
    // ---- s3 (N3 > 1)
    __device__ static __forceinline__ void s3_ld(float2 *v, const float2 *sm, const TW &tw) {
#pragma unroll
        for (int i = 0; i < L::B2; ++i)
#pragma unroll
            for (int k2 = 0; k2 < N2; ++k2) {
                float2 a = sm[tw.slotB(i, k2)];
                if (k2 > 0) a = cmulc(a, tw.w2at(i, k2));
                v[i * N2 + k2] = a;
            }
    }
    __device__ static __forceinline__ void s3_a(float2 *v) {
#pragma unroll
        for (int i = 0; i < L::B2; ++i) dftR<N2, +1>(v + i * N2);
    }
    __device__ static __forceinline__ void s3_st(const float2 *v, float2 *sm, const TW &tw) {
#pragma unroll
        for (int i = 0; i < L::B2; ++i)
#pragma unroll
            for (int n2 = 0; n2 < N2; ++n2) sm[tw.slotB(i, n2)] = v[i * N2 + n2];
    }
    // ---- s4
    __device__ static __forceinline__ void s4_ld(float2 *v, const float2 *sm, const TW &tw) {
#pragma unroll
        for (int i = 0; i < L::B1; ++i)
#pragma unroll
            for (int k1 = 0; k1 < N1; ++k1) {
                float2 a = sm[tw.slotA(i, k1)];
                if (k1 > 0) a = cmulc(a, tw.w1[i][k1]);
                v[i * N1 + k1] = (HALF && (k1 & 1)) ? make_float2(-a.x, -a.y) : a;
            }
    }
    __device__ static __forceinline__ void s4_a(float2 *v) {
#pragma unroll
        for (int i = 0; i < L::B1; ++i) dftR<N1, +1>(v + i * N1);
    }
    // N = 16: one thread holds the whole line in natural order, u = q
    __device__ static __forceinline__ void mask16(float2 *v, const float2 *__restrict__ gperm) {
#pragma unroll
        for (int q = 0; q < N1; ++q) {
            if (HALF) v[q] = ((q & 1) != (q >= N / 2)) ? make_float2(-v[q].x, -v[q].y) : v[q];
            else v[q] = cmul(v[q], __ldg(&gperm[q]));
        }
    }

    // ---------------- forward half only (general 2-D masks): on return v[i*RL + q] is position
    // p = (t + TPL*i)*RL + q of the digit-reversed spectrum (un-normalised).  The barrier on
    // entry separates it from whatever used the exchange line before.
    __device__ static __forceinline__ void forward(float2 *v, float2 *sm, int t, int group, const TW &tw) {
        s0_a(v);
        if (N2 > 1) {
            group_sync<TPL>(group);
            s0_b(v, sm, tw);
            group_sync<TPL>(group);
            if (N3 > 1) {
                s1_ld(v, sm, tw);
                s1_a(v);
                s1_b(v, sm, tw);
                group_sync<TPL>(group);
            }
            s2_ld(v, sm, tw);
            s2_a(v);
        }
    }
    // ---------------- inverse half only, from that layout to natural order (un-normalised)
    __device__ static __forceinline__ void inverse(float2 *v, float2 *sm, int t, int group, const TW &tw) {
        static_assert(!HALF, "inverse() is the plain inverse transform");
        if (N2 > 1) {
#pragma unroll
            for (int i = 0; i < L::BL; ++i) dftR<RL, +1>(v + i * RL);
            group_sync<TPL>(group);
            s2_st(v, sm, tw);
            group_sync<TPL>(group);
            if (N3 > 1) {
                s3_ld(v, sm, tw);
                s3_a(v);
                s3_st(v, sm, tw);
                group_sync<TPL>(group);
            }
            s4_ld(v, sm, tw);
        }
        s4_a(v);
    }

    // ---------------- one line
    __device__ static __forceinline__ void run(float2 *v, float2 *sm, int t, int group, const TW &tw,
                                               const float2 *__restrict__ gperm) {
        s0_a(v);
        if (N2 == 1) {
            mask16(v, gperm);
        } else {
            s0_b(v, sm, tw);
            group_sync<TPL>(group);
            if (N3 > 1) {
                s1_ld(v, sm, tw);
                s1_a(v);
                s1_b(v, sm, tw);
                group_sync<TPL>(group);
            }
            s2_ld(v, sm, tw);
            s2_a(v);
            s2_b(v, t, tw, gperm);
            s2_st(v, sm, tw);
            group_sync<TPL>(group);
            if (N3 > 1) {
                s3_ld(v, sm, tw);
                s3_a(v);
                s3_st(v, sm, tw);
                group_sync<TPL>(group);
            }
            s4_ld(v, sm, tw);
        }
        s4_a(v);
    }
};

}  // namespace pyr
