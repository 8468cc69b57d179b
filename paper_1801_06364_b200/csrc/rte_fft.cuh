// rte_fft.cuh — register-resident complex DFTs of small fixed size for the pencil-FFT kernels (sm_100a).
//
// The spectral derivative of PAPER.md eq.(7)-(8),(10) needs DFT_n / IDFT_n along a pencil with
// n = N1*N2.  Each thread computes whole N1- or N2-point transforms in registers; everything here is fully
// unrolled at compile time, twiddle factors are compile-time immediates (FFMA/FMUL immediate forms), and the
// "natural order in, natural order out" contract makes the index bookkeeping of the callers trivial (the output
// permutation of the Cooley-Tukey split is a register renaming, i.e. free).
//
// Forward sign: X[k] = sum_j x[j] exp(-2 pi i j k / R)   (eq.(8): exp(-i k.r)).
// Inverse (unnormalised): the same butterflies with conjugated twiddles (template flag INV).
#pragma once
#include <cuda_runtime.h>
#include <math.h>

#ifndef RTE_HD
#define RTE_HD __host__ __device__ __forceinline__
#endif

namespace rtefft {

// ---- compile-time cos/sin of 2 pi num/den (double precision Taylor series after octant reduction) ---------------
constexpr double kTwoPi = 6.283185307179586476925286766559005768;

__host__ __device__ constexpr double taylor_sin(double x) {  // |x| <= pi/4
    double x2 = x * x, term = x, sum = x;
    for (int i = 1; i < 14; ++i) { term *= -x2 / (double)((2 * i) * (2 * i + 1)); sum += term; }
    return sum;
}
__host__ __device__ constexpr double taylor_cos(double x) {  // |x| <= pi/4
    double x2 = x * x, term = 1.0, sum = 1.0;
    for (int i = 1; i < 14; ++i) { term *= -x2 / (double)((2 * i - 1) * (2 * i)); sum += term; }
    return sum;
}
// cos(2 pi f) for f in [0,1)
__host__ __device__ constexpr double cos_turn(double f) {
    if (f > 0.5) f = 1.0 - f;                   // cos symmetric about half a turn
    if (f > 0.25) return -cos_turn(0.5 - f);    // second quadrant
    if (f <= 0.125) return taylor_cos(kTwoPi * f);
    return taylor_sin(kTwoPi * (0.25 - f));
}
__host__ __device__ constexpr double cos2pi(int num, int den) {
    int r = ((num % den) + den) % den;
    return cos_turn((double)r / (double)den);
}
__host__ __device__ constexpr double sin2pi(int num, int den) {    // sin(2 pi x) = cos(2 pi (x - 1/4))
    return cos2pi(4 * num - den, 4 * den);
}

// ---- packed complex arithmetic ----------------------------------------------------------------------------------------
// A complex number is one float2 = one aligned 64-bit register pair.  sm_100a has packed fp32 instructions
// (PTX add/mul/fma.rn.f32x2 -> SASS FADD2/FMUL2/FFMA2) that do both halves in ONE issue slot, and ptxas folds the
// half-swap, the per-half negation and the scalar broadcast of the operands below into operand modifiers
// (.LO_HI, .NP, .F32), so a complex add is 1 instruction and a complex-by-constant multiply is 2 (scalar: 2 and 4).
// Same IEEE roundings as the scalar forms (each half is an independent fp32 add / mul / fma).
#ifdef __CUDA_ARCH__
typedef unsigned long long c64_t;
__device__ __forceinline__ c64_t pk(float lo, float hi) { c64_t r; asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ float2 up(c64_t v) { float2 r; asm("mov.b64 {%0,%1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(v)); return r; }
__device__ __forceinline__ c64_t add2(c64_t a, c64_t b) { c64_t d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ c64_t mul2(c64_t a, c64_t b) { c64_t d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ c64_t fma2(c64_t a, c64_t b, c64_t c) { c64_t d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
#define RTE_PACKED(packed_expr, scalar_expr) return packed_expr
#else
#define RTE_PACKED(packed_expr, scalar_expr) return scalar_expr
#endif
RTE_HD float2 cadd(float2 a, float2 b) { RTE_PACKED(up(add2(pk(a.x, a.y), pk(b.x, b.y))), make_float2(a.x + b.x, a.y + b.y)); }
RTE_HD float2 csub(float2 a, float2 b) { RTE_PACKED(up(add2(pk(a.x, a.y), pk(-b.x, -b.y))), make_float2(a.x - b.x, a.y - b.y)); }
RTE_HD float2 cadd_mi(float2 a, float2 b) {   // a - i b
    RTE_PACKED(up(add2(pk(a.x, a.y), pk(b.y, -b.x))), make_float2(a.x + b.y, a.y - b.x));
}
RTE_HD float2 cadd_pi(float2 a, float2 b) {   // a + i b
    RTE_PACKED(up(add2(pk(a.x, a.y), pk(-b.y, b.x))), make_float2(a.x - b.y, a.y + b.x));
}
RTE_HD float2 cscale(float2 a, float s) { RTE_PACKED(up(mul2(pk(a.x, a.y), pk(s, s))), make_float2(a.x * s, a.y * s)); }
RTE_HD float2 cmul_cs(float2 a, float c, float s) {   // a * (c - i s) = c (a.x, a.y) + s (a.y, -a.x)
    RTE_PACKED(up(fma2(pk(a.y, -a.x), pk(s, s), mul2(pk(a.x, a.y), pk(c, c)))),
               make_float2(fmaf(a.y, s, a.x * c), fmaf(-a.x, s, a.y * c)));
}
RTE_HD float2 cmul(float2 a, float2 w) {   // a * w = w.x (a.x, a.y) + w.y (-a.y, a.x)
    RTE_PACKED(up(fma2(pk(-a.y, a.x), pk(w.y, w.y), mul2(pk(a.x, a.y), pk(w.x, w.x)))),
               make_float2(fmaf(-a.y, w.y, a.x * w.x), fmaf(a.x, w.y, a.y * w.x)));
}
RTE_HD float2 cmulc(float2 a, float2 w) {  // a * conj(w) = w.x (a.x, a.y) + w.y (a.y, -a.x)
    RTE_PACKED(up(fma2(pk(a.y, -a.x), pk(w.y, w.y), mul2(pk(a.x, a.y), pk(w.x, w.x)))),
               make_float2(fmaf(a.y, w.y, a.x * w.x), fmaf(-a.x, w.y, a.y * w.x)));
}
RTE_HD float2 caxpy(float s, float2 a, float2 acc) {   // acc + s * a (both halves)
    RTE_PACKED(up(fma2(pk(s, s), pk(a.x, a.y), pk(acc.x, acc.y))), make_float2(fmaf(s, a.x, acc.x), fmaf(s, a.y, acc.y)));
}
// acc + (wx * a.x, wy * a.y): the diagonal part of a 2x2 real block applied to a pair
RTE_HD float2 cfma_diag(float wx, float wy, float2 a, float2 acc) {
    RTE_PACKED(up(fma2(pk(wx, wy), pk(a.x, a.y), pk(acc.x, acc.y))), make_float2(fmaf(wx, a.x, acc.x), fmaf(wy, a.y, acc.y)));
}
// acc + (wx * a.y, wy * a.x): the off-diagonal part
RTE_HD float2 cfma_swap(float wx, float wy, float2 a, float2 acc) {
    RTE_PACKED(up(fma2(pk(wx, wy), pk(a.y, a.x), pk(acc.x, acc.y))), make_float2(fmaf(wx, a.y, acc.x), fmaf(wy, a.x, acc.y)));
}

// a * exp(-2 pi i NUM/DEN) with the multiples of an eighth turn special-cased
template <int NUM, int DEN>
RTE_HD float2 mulw(float2 a) {
    constexpr int r = ((NUM % DEN) + DEN) % DEN;
    constexpr float h = 0.70710678118654752440f;
    if constexpr (r == 0) return a;
    else if constexpr (4 * r == DEN) return make_float2(a.y, -a.x);                       // * -i
    else if constexpr (2 * r == DEN) return make_float2(-a.x, -a.y);                      // * -1
    else if constexpr (4 * r == 3 * DEN) return make_float2(-a.y, a.x);                   // * +i
    else if constexpr (8 * r == DEN) return cscale(cadd_mi(a, a), h);                     // (1-i)/sqrt2:  h (a - i a)
    else if constexpr (8 * r == 3 * DEN) return cscale(cadd_pi(a, a), -h);                // (-1-i)/sqrt2: -h (a + i a)
    else if constexpr (8 * r == 5 * DEN) return cscale(cadd_mi(a, a), -h);                // (-1+i)/sqrt2: -h (a - i a)
    else if constexpr (8 * r == 7 * DEN) return cscale(cadd_pi(a, a), h);                 // (1+i)/sqrt2:  h (a + i a)
    else {
        constexpr float c = (float)cos2pi(r, DEN);
        constexpr float s = (float)sin2pi(r, DEN);   // w = c - i s
        return cmul_cs(a, c, s);
    }
}

// ---- DFT of R points held at v[0], v[S], v[2S], ...; natural order in and out --------------------------------------
// INV = false: X[k] = sum_j x[j] exp(-2 pi i j k / R); INV = true: the unnormalised inverse, exp(+2 pi i j k / R) — the
// same butterflies with every twiddle conjugated (no re/im swaps of the data, so results are born in the register
// pairs the stores and reductions need).
template <int R, int S, bool INV>
struct Dft;

template <int S, bool INV>
struct Dft<1, S, INV> {
    static RTE_HD void run(float2*) {}
};

template <int S, bool INV>
struct Dft<2, S, INV> {
    static RTE_HD void run(float2* v) {
        const float2 a = v[0], b = v[S];
        v[0] = cadd(a, b);
        v[S] = csub(a, b);
    }
};

template <int S, bool INV>
struct Dft<3, S, INV> {
    static RTE_HD void run(float2* v) {
        constexpr float hs3 = INV ? -0.86602540378443864676f : 0.86602540378443864676f;   // -+ sqrt(3)/2
        const float2 a = v[0], b = v[S], c = v[2 * S];
        const float2 s = cadd(b, c), d = csub(b, c);
        const float2 m = caxpy(-0.5f, s, a);
        // forward: X1 = m - i hs3 d ; X2 = m + i hs3 d   (inverse: the conjugate twiddles swap the two)
        v[0] = cadd(a, s);
        v[S] = caxpy(hs3, make_float2(d.y, -d.x), m);
        v[2 * S] = caxpy(hs3, make_float2(-d.y, d.x), m);
    }
};

template <int S, bool INV>
struct Dft<4, S, INV> {
    static RTE_HD void run(float2* v) {
        const float2 a = v[0], b = v[S], c = v[2 * S], d = v[3 * S];
        const float2 t0 = cadd(a, c), t1 = csub(a, c), t2 = cadd(b, d), t3 = csub(b, d);
        v[0] = cadd(t0, t2);
        v[2 * S] = csub(t0, t2);
        v[S] = INV ? cadd_pi(t1, t3) : cadd_mi(t1, t3);       // t1 -+ i t3
        v[3 * S] = INV ? cadd_mi(t1, t3) : cadd_pi(t1, t3);   // t1 +- i t3
    }
};

// first factor of the Cooley-Tukey split R = RA * RB
template <int R>
struct Split {
    static constexpr int RA = (R % 3 == 0) ? 3 : ((R == 8) ? 2 : ((R % 4 == 0) ? 4 : 2));
    static constexpr int RB = R / RA;
};

template <int RA, int RB, int S, int KA, int B, bool INV>
struct TwiddleRow {   // v[(RB*KA + b)*S] *= W_R^{+-b*KA} for b = B..RB-1
    static RTE_HD void run(float2* v) {
        if constexpr (B < RB) {
            v[(RB * KA + B) * S] = mulw<(INV ? -B * KA : B * KA), RA * RB>(v[(RB * KA + B) * S]);
            TwiddleRow<RA, RB, S, KA, B + 1, INV>::run(v);
        }
    }
};
template <int RA, int RB, int S, int KA, bool INV>
struct TwiddleAll {
    static RTE_HD void run(float2* v) {
        if constexpr (KA < RA) {
            TwiddleRow<RA, RB, S, KA, 1, INV>::run(v);
            TwiddleAll<RA, RB, S, KA + 1, INV>::run(v);
        }
    }
};

// generic: x[j], j = RB*a + b ; X[ka + RA*kb]
//   step 1: for each b, DFT_RA over a (stride RB*S)          -> slot (RB*ka + b) holds Y[ka][b]
//   step 2: slot (RB*ka + b) *= W_R^{b ka}
//   step 3: for each ka, DFT_RB over b (stride S)             -> slot (RB*ka + kb) holds X[ka + RA*kb]
//   step 4: un-permute (register renaming)
template <int R, int S, bool INV>
struct Dft {
    static constexpr int RA = Split<R>::RA, RB = Split<R>::RB;
    static RTE_HD void run(float2* v) {
#pragma unroll
        for (int b = 0; b < RB; ++b) Dft<RA, RB * S, INV>::run(v + b * S);
        TwiddleAll<RA, RB, S, 1, INV>::run(v);
#pragma unroll
        for (int ka = 0; ka < RA; ++ka) Dft<RB, S, INV>::run(v + ka * RB * S);
        float2 t[R];
#pragma unroll
        for (int ka = 0; ka < RA; ++ka)
#pragma unroll
            for (int kb = 0; kb < RB; ++kb) t[ka + RA * kb] = v[(RB * ka + kb) * S];
#pragma unroll
        for (int k = 0; k < R; ++k) v[k * S] = t[k];
    }
};

template <int R>
RTE_HD void dft_fwd(float2 (&v)[R]) {
    Dft<R, 1, false>::run(v);
}
template <int R>
RTE_HD void dft_inv(float2 (&v)[R]) {   // unnormalised inverse
    Dft<R, 1, true>::run(v);
}

// The same inverse as swap(re,im) o forward o swap(re,im).  Needs two register moves per output when the result
// feeds a store (the half-swap cannot fold into a store operand) but a few registers fewer than dft_inv; the x pass,
// whose tail also holds the re-read psi column, uses it to stay spill-free at 128 registers.
template <int R>
RTE_HD void dft_inv_swap(float2 (&v)[R]) {
#pragma unroll
    for (int i = 0; i < R; ++i) { const float t = v[i].x; v[i].x = v[i].y; v[i].y = t; }
    Dft<R, 1, false>::run(v);
#pragma unroll
    for (int i = 0; i < R; ++i) { const float t = v[i].x; v[i].x = v[i].y; v[i].y = t; }
}

}  // namespace rtefft
