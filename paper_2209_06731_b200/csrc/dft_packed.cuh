// dft_packed.cuh -- small complex DFTs in registers on TWO transforms at once, packed FP32 (sm_100a).
//
// Blackwell's FP32 pipe executes add/mul/fma.f32x2 (SASS FADD2/FMUL2/FFMA2) at the scalar lane rate in half
// the issue slots (bench.py --ubench).  A pk::c2 carries the real parts of two complex numbers ("lane 0" and
// "lane 1") in one 64-bit register pair and their imaginary parts in another (planar form), so that every
// complex operation -- including multiplication by i and by a twiddle shared by both lanes -- is made of
// packed instructions only.  The kernels of nl_rx_kernels.cuh choose the two lanes so that both transforms
// share addresses, twiddles and zero patterns:
//   * inverse x passes:  lane 0 = i kx f,  lane 1 = i ky f   of the same column (d_x and d_y of one field);
//   * inverse y (row):   lane 0 / lane 1 = the two real fields d_x f, d_y f (two C2R transforms);
//   * forward x passes:  two neighbouring ky columns.
//
// Everything is __host__ __device__: tests/host_emul compiles the same functions for the CPU (the packed
// operations fall back to two scalar operations there) and runs the kernels' phases thread by thread.
//
// dft<N,S,ZM>(v): v[0..N-1] (natural order) <- DFT, X[k] = sum_n v[n] e^{S 2 pi i n k / N}, lane-wise.
// N in {2,3,4,6,8,12,16,32}.  ZM: bit n set <=> v[n] is known to be zero (2/3-rule padding).
#pragma once
#include <cuda_runtime.h>

#include <cstring>

#include "dft_regs.cuh"   // cos192 / sin192 constant tables, zm_t, sub_mask_first/second

#ifndef GX_HD
#define GX_HD __host__ __device__ __forceinline__
#endif

namespace gx {
namespace pk {

typedef unsigned long long u64;
struct c2 { u64 re, im; };

GX_HD u64 pk2(float a, float b) {
#ifdef __CUDA_ARCH__
    u64 r; asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(a), "f"(b)); return r;
#else
    unsigned ua, ub; std::memcpy(&ua, &a, 4); std::memcpy(&ub, &b, 4); return (u64)ua | ((u64)ub << 32);
#endif
}
GX_HD void upk2(u64 v, float& a, float& b) {
#ifdef __CUDA_ARCH__
    asm("mov.b64 {%0,%1}, %2;" : "=f"(a), "=f"(b) : "l"(v));
#else
    unsigned ua = (unsigned)(v & 0xffffffffull), ub = (unsigned)(v >> 32);
    std::memcpy(&a, &ua, 4); std::memcpy(&b, &ub, 4);
#endif
}
GX_HD float lo(u64 v) { float a, b; upk2(v, a, b); return a; }
GX_HD float hi(u64 v) { float a, b; upk2(v, a, b); return b; }
GX_HD u64 bc2(float s) { return pk2(s, s); }
GX_HD u64 add2(u64 a, u64 b) {
#ifdef __CUDA_ARCH__
    u64 r; asm("add.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r;
#else
    return pk2(lo(a) + lo(b), hi(a) + hi(b));
#endif
}
GX_HD u64 sub2(u64 a, u64 b) {
#ifdef __CUDA_ARCH__
    u64 r; asm("sub.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r;
#else
    return pk2(lo(a) - lo(b), hi(a) - hi(b));
#endif
}
GX_HD u64 mul2(u64 a, u64 b) {
#ifdef __CUDA_ARCH__
    u64 r; asm("mul.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r;
#else
    return pk2(lo(a) * lo(b), hi(a) * hi(b));
#endif
}
GX_HD u64 fma2(u64 a, u64 b, u64 c) {
#ifdef __CUDA_ARCH__
    u64 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r;
#else
    return pk2(fmaf(lo(a), lo(b), lo(c)), fmaf(hi(a), hi(b), hi(c)));
#endif
}
GX_HD u64 neg2(u64 a) { return a ^ 0x8000000080000000ull; }

GX_HD c2 make_c2(u64 re, u64 im) { c2 r; r.re = re; r.im = im; return r; }
GX_HD c2 czero() { return make_c2(0ull, 0ull); }
GX_HD c2 cadd(c2 a, c2 b) { return make_c2(add2(a.re, b.re), add2(a.im, b.im)); }
GX_HD c2 csub(c2 a, c2 b) { return make_c2(sub2(a.re, b.re), sub2(a.im, b.im)); }
GX_HD c2 cneg(c2 a) { return make_c2(neg2(a.re), neg2(a.im)); }
GX_HD c2 conj(c2 a) { return make_c2(a.re, neg2(a.im)); }
// a * (c + i s), the same scalar factor on both lanes
GX_HD c2 cmul_s(c2 a, float c, float s) {
    return make_c2(fma2(a.im, bc2(-s), mul2(a.re, bc2(c))), fma2(a.re, bc2(s), mul2(a.im, bc2(c))));
}
// conj(a) * (c + i s)
GX_HD c2 cmul_conj_s(c2 a, float c, float s) {
    return make_c2(fma2(a.im, bc2(s), mul2(a.re, bc2(c))), fma2(a.re, bc2(s), mul2(a.im, bc2(-c))));
}
template <int S> GX_HD c2 mul_i(c2 a) {   // a * (S i)
    return S > 0 ? make_c2(neg2(a.im), a.re) : make_c2(a.im, neg2(a.re));
}
// b + (S i) d  and  b - (S i) d  without materialising the rotation
template <int S> GX_HD void rot_pm(c2 b, c2 d, c2& plus, c2& minus) {
    if (S > 0) {
        plus = make_c2(sub2(b.re, d.im), add2(b.im, d.re));
        minus = make_c2(add2(b.re, d.im), sub2(b.im, d.re));
    } else {
        plus = make_c2(add2(b.re, d.im), sub2(b.im, d.re));
        minus = make_c2(sub2(b.re, d.im), add2(b.im, d.re));
    }
}

// v * e^{S 2 pi i t / N}, t and N compile-time after unrolling (N | 192)
template <int N, int S> GX_HD c2 twiddle(c2 v, int t) {
    static_assert(192 % N == 0, "N must divide 192");
    const int a = ((t * (192 / N)) % 192 + 192) % 192;
    if (a == 0) return v;
    if (a == 48) return mul_i<S>(v);
    if (a == 96) return cneg(v);
    if (a == 144) return mul_i<-S>(v);
    const float c = (float)cos192(a);
    const float s = (float)sin192(a) * (S > 0 ? 1.f : -1.f);
    return cmul_s(v, c, s);
}

template <int N, int S, zm_t ZM = 0ull> struct Dft;

template <int S, zm_t ZM> struct Dft<2, S, ZM> {
    GX_HD static void run(c2 (&v)[2]) {
        constexpr bool z0 = ZM & 1u, z1 = ZM & 2u;
        const c2 a = v[0], b = v[1];
        if constexpr (z1) { v[1] = a; }
        else if constexpr (z0) { v[0] = b; v[1] = cneg(b); }
        else { v[0] = cadd(a, b); v[1] = csub(a, b); }
    }
};

template <int S, zm_t ZM> struct Dft<3, S, ZM> {
    GX_HD static void run(c2 (&v)[3]) {
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

template <int S, zm_t ZM> struct Dft<4, S, ZM> {
    GX_HD static void run(c2 (&v)[4]) {
        constexpr bool z0 = ZM & 1u, z1 = ZM & 2u, z2 = ZM & 4u, z3 = ZM & 8u;
        c2 a, b, c, d;                                    // a = v0+v2, b = v0-v2, c = v1+v3, d = v1-v3
        if constexpr (z2) { a = v[0]; b = v[0]; }
        else if constexpr (z0) { a = v[2]; b = cneg(v[2]); }
        else { a = cadd(v[0], v[2]); b = csub(v[0], v[2]); }
        if constexpr (z3) { c = v[1]; d = v[1]; }
        else if constexpr (z1) { c = v[3]; d = cneg(v[3]); }
        else { c = cadd(v[1], v[3]); d = csub(v[1], v[3]); }
        if constexpr (z1 && z3) { v[0] = a; v[1] = b; v[2] = a; v[3] = b; }
        else if constexpr (z0 && z2) { const c2 e = mul_i<S>(d); v[0] = c; v[1] = e; v[2] = cneg(c); v[3] = cneg(e); }
        else { v[0] = cadd(a, c); v[2] = csub(a, c); rot_pm<S>(b, d, v[1], v[3]); }
    }
};

// One Cooley-Tukey split N = A*B:  n = n1*B + n2,  k = k1 + A*k2.
template <int N, int A, int B, int S, zm_t ZM, int n2>
GX_HD void dft_split_col(const c2 (&v)[N], c2 (&y)[N]) {
    c2 t[A];
#pragma unroll
    for (int n1 = 0; n1 < A; ++n1) t[n1] = v[n1 * B + n2];
    Dft<A, S, sub_mask_first<A, B, ZM, n2>()>::run(t);
#pragma unroll
    for (int k1 = 0; k1 < A; ++k1) y[k1 * B + n2] = twiddle<N, S>(t[k1], n2 * k1);
    if constexpr (n2 + 1 < B) dft_split_col<N, A, B, S, ZM, n2 + 1>(v, y);
}

template <int N, int A, int B, int S, zm_t ZM = 0ull> GX_HD void dft_split(c2 (&v)[N]) {
    static_assert(A * B == N, "bad split");
    c2 y[N];
    dft_split_col<N, A, B, S, ZM, 0>(v, y);
#pragma unroll
    for (int k1 = 0; k1 < A; ++k1) {
        c2 u[B];
#pragma unroll
        for (int n2 = 0; n2 < B; ++n2) u[n2] = y[k1 * B + n2];
        Dft<B, S, sub_mask_second<A, B, ZM>()>::run(u);
#pragma unroll
        for (int k2 = 0; k2 < B; ++k2) v[k1 + A * k2] = u[k2];
    }
}

template <int S, zm_t ZM> struct Dft<6, S, ZM> {
    GX_HD static void run(c2 (&v)[6]) { dft_split<6, 2, 3, S, ZM>(v); }
};
template <int S, zm_t ZM> struct Dft<8, S, ZM> {
    GX_HD static void run(c2 (&v)[8]) { dft_split<8, 2, 4, S, ZM>(v); }
};
template <int S, zm_t ZM> struct Dft<12, S, ZM> {
    GX_HD static void run(c2 (&v)[12]) { dft_split<12, 3, 4, S, ZM>(v); }
};
template <int S, zm_t ZM> struct Dft<16, S, ZM> {
    GX_HD static void run(c2 (&v)[16]) { dft_split<16, 4, 4, S, ZM>(v); }
};
template <int S, zm_t ZM> struct Dft<32, S, ZM> {
    GX_HD static void run(c2 (&v)[32]) { dft_split<32, 4, 8, S, ZM>(v); }
};

template <int N, int S, zm_t ZM = 0ull> GX_HD void dft(c2 (&v)[N]) { Dft<N, S, ZM>::run(v); }

}  // namespace pk
}  // namespace gx
