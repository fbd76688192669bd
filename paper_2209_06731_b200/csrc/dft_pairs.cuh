// dft_pairs.cuh -- small complex DFTs in registers on TWO independent transforms at once (sm_100a).
//
// Blackwell's FP32 pipe executes the packed instructions FADD2 / FMUL2 / FFMA2 (PTX add/mul/fma.f32x2)
// at the same lane rate as the scalar forms but with half the issue slots (profiles/r01_ubench_fp32_pipe.txt).
// The butterflies of the FFT passes are issue-bound in scalar form (profiles/r01a_bracket_ncu_full.md), so
// every value here is a pair: c2 holds the real parts of two unrelated complex numbers in one 64-bit
// register pair and their imaginary parts in another ("lane a" and "lane b": two ky columns in the x
// passes, two x rows in the y passes).  Twiddles are shared by both lanes and enter as scalars, which
// ptxas encodes as the broadcast operand form (R.F32 / immediate) of the packed instructions.
//
// dft2<N,S,ZM>(v): v[0..N-1] (natural order) <- DFT, X[k] = sum_n v[n] e^{S 2 pi i n k / N}, lane-wise.
// N in {2,3,4,6,8,12,16}.  ZM: bit n set <=> v[n] is known to be zero (2/3-rule padding).
#pragma once
#include <cuda_runtime.h>

#include "dft_regs.cuh"   // cos48 / sin48 constant tables

namespace gx {

typedef unsigned long long u64;
struct c2 { u64 re, im; };

__device__ __forceinline__ u64 pk2(float a, float b) { u64 r; asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ void upk2(u64 v, float& a, float& b) { asm("mov.b64 {%0,%1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); }
__device__ __forceinline__ u64 bc2(float s) { return pk2(s, s); }
__device__ __forceinline__ u64 add2(u64 a, u64 b) { u64 r; asm("add.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 sub2(u64 a, u64 b) { u64 r; asm("sub.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 mul2(u64 a, u64 b) { u64 r; asm("mul.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) { u64 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ u64 neg2(u64 a) { return a ^ 0x8000000080000000ull; }

__device__ __forceinline__ c2 czero2() { c2 r; r.re = 0ull; r.im = 0ull; return r; }
__device__ __forceinline__ c2 cadd(c2 a, c2 b) { c2 r; r.re = add2(a.re, b.re); r.im = add2(a.im, b.im); return r; }
__device__ __forceinline__ c2 csub(c2 a, c2 b) { c2 r; r.re = sub2(a.re, b.re); r.im = sub2(a.im, b.im); return r; }
__device__ __forceinline__ c2 cneg(c2 a) { c2 r; r.re = neg2(a.re); r.im = neg2(a.im); return r; }
// a * (c + i s), the same scalar twiddle on both lanes
__device__ __forceinline__ c2 cmul_s(c2 a, float c, float s) {
    c2 r;
    r.re = fma2(a.im, bc2(-s), mul2(a.re, bc2(c)));
    r.im = fma2(a.re, bc2(s), mul2(a.im, bc2(c)));
    return r;
}
template <int S> __device__ __forceinline__ c2 mul_i2(c2 a) {   // a * (S i)
    c2 r;
    if (S > 0) { r.re = neg2(a.im); r.im = a.re; } else { r.re = a.im; r.im = neg2(a.re); }
    return r;
}
// b + (S i) d  and  b - (S i) d  without materialising the rotation
template <int S> __device__ __forceinline__ void rot_pm(c2 b, c2 d, c2& plus, c2& minus) {
    if (S > 0) {
        plus.re = sub2(b.re, d.im); plus.im = add2(b.im, d.re);
        minus.re = add2(b.re, d.im); minus.im = sub2(b.im, d.re);
    } else {
        plus.re = add2(b.re, d.im); plus.im = sub2(b.im, d.re);
        minus.re = sub2(b.re, d.im); minus.im = add2(b.im, d.re);
    }
}

// v * e^{S 2 pi i t / N}, t and N compile-time after unrolling
template <int N, int S> __device__ __forceinline__ c2 twiddle2(c2 v, int t) {
    static_assert(48 % N == 0, "N must divide 48");
    const int a = ((t * (48 / N)) % 48 + 48) % 48;
    if (a == 0) return v;
    if (a == 12) return mul_i2<S>(v);
    if (a == 24) return cneg(v);
    if (a == 36) return mul_i2<-S>(v);
    const float c = (float)cos48(a);
    const float s = (float)sin48(a) * (S > 0 ? 1.f : -1.f);
    return cmul_s(v, c, s);
}

template <int N, int S, zm_t ZM = 0ull> struct Dft2;

template <int S, zm_t ZM> struct Dft2<2, S, ZM> {
    __device__ __forceinline__ static void run(c2 (&v)[2]) {
        constexpr bool z0 = ZM & 1u, z1 = ZM & 2u;
        const c2 a = v[0], b = v[1];
        if constexpr (z1) { v[1] = a; }
        else if constexpr (z0) { v[0] = b; v[1] = cneg(b); }
        else { v[0] = cadd(a, b); v[1] = csub(a, b); }
    }
};

template <int S, zm_t ZM> struct Dft2<3, S, ZM> {
    __device__ __forceinline__ static void run(c2 (&v)[3]) {
        const c2 t = cadd(v[1], v[2]);
        const c2 d = csub(v[1], v[2]);
        c2 m;
        m.re = fma2(t.re, bc2(-0.5f), v[0].re);
        m.im = fma2(t.im, bc2(-0.5f), v[0].im);
        constexpr float h = 0.86602540378443864676f * (S > 0 ? 1.f : -1.f);
        v[0] = cadd(v[0], t);
        // r = (S i) |h| d :  v1 = m + r, v2 = m - r
        v[1].re = fma2(d.im, bc2(-h), m.re); v[1].im = fma2(d.re, bc2(h), m.im);
        v[2].re = fma2(d.im, bc2(h), m.re);  v[2].im = fma2(d.re, bc2(-h), m.im);
    }
};

template <int S, zm_t ZM> struct Dft2<4, S, ZM> {
    __device__ __forceinline__ static void run(c2 (&v)[4]) {
        constexpr bool z0 = ZM & 1u, z1 = ZM & 2u, z2 = ZM & 4u, z3 = ZM & 8u;
        c2 a, b, c, d;                                    // a = v0+v2, b = v0-v2, c = v1+v3, d = v1-v3
        if constexpr (z2) { a = v[0]; b = v[0]; }
        else if constexpr (z0) { a = v[2]; b = cneg(v[2]); }
        else { a = cadd(v[0], v[2]); b = csub(v[0], v[2]); }
        if constexpr (z3) { c = v[1]; d = v[1]; }
        else if constexpr (z1) { c = v[3]; d = cneg(v[3]); }
        else { c = cadd(v[1], v[3]); d = csub(v[1], v[3]); }
        if constexpr (z1 && z3) { v[0] = a; v[1] = b; v[2] = a; v[3] = b; }
        else if constexpr (z0 && z2) { const c2 e = mul_i2<S>(d); v[0] = c; v[1] = e; v[2] = cneg(c); v[3] = cneg(e); }
        else { v[0] = cadd(a, c); v[2] = csub(a, c); rot_pm<S>(b, d, v[1], v[3]); }
    }
};

template <int N, int A, int B, int S, zm_t ZM, int n2>
__device__ __forceinline__ void dft2_split_col(const c2 (&v)[N], c2 (&y)[N]) {
    c2 t[A];
#pragma unroll
    for (int n1 = 0; n1 < A; ++n1) t[n1] = v[n1 * B + n2];
    Dft2<A, S, sub_mask_first<A, B, ZM, n2>()>::run(t);
#pragma unroll
    for (int k1 = 0; k1 < A; ++k1) y[k1 * B + n2] = twiddle2<N, S>(t[k1], n2 * k1);
    if constexpr (n2 + 1 < B) dft2_split_col<N, A, B, S, ZM, n2 + 1>(v, y);
}

template <int N, int A, int B, int S, zm_t ZM = 0ull> __device__ __forceinline__ void dft2_split(c2 (&v)[N]) {
    static_assert(A * B == N, "bad split");
    c2 y[N];
    dft2_split_col<N, A, B, S, ZM, 0>(v, y);
#pragma unroll
    for (int k1 = 0; k1 < A; ++k1) {
        c2 u[B];
#pragma unroll
        for (int n2 = 0; n2 < B; ++n2) u[n2] = y[k1 * B + n2];
        Dft2<B, S, sub_mask_second<A, B, ZM>()>::run(u);
#pragma unroll
        for (int k2 = 0; k2 < B; ++k2) v[k1 + A * k2] = u[k2];
    }
}

template <int S, zm_t ZM> struct Dft2<6, S, ZM> {
    __device__ __forceinline__ static void run(c2 (&v)[6]) { dft2_split<6, 2, 3, S, ZM>(v); }
};
template <int S, zm_t ZM> struct Dft2<8, S, ZM> {
    __device__ __forceinline__ static void run(c2 (&v)[8]) { dft2_split<8, 2, 4, S, ZM>(v); }
};
template <int S, zm_t ZM> struct Dft2<12, S, ZM> {
    __device__ __forceinline__ static void run(c2 (&v)[12]) { dft2_split<12, 3, 4, S, ZM>(v); }
};
template <int S, zm_t ZM> struct Dft2<16, S, ZM> {
    __device__ __forceinline__ static void run(c2 (&v)[16]) { dft2_split<16, 4, 4, S, ZM>(v); }
};

template <int N, int S, zm_t ZM = 0ull> __device__ __forceinline__ void dft2(c2 (&v)[N]) { Dft2<N, S, ZM>::run(v); }

}  // namespace gx
