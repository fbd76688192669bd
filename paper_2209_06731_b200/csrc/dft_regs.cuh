// dft_regs.cuh -- small complex DFTs held entirely in registers (sm_100a, fp32).
//
// Building block of the shared-memory FFT passes in nl_kernels.cuh.  dft<N,S>(v) overwrites the
// N complex values v[0..N-1] (natural order) with their DFT, X[k] = sum_n v[n] e^{S 2 pi i n k / N},
// S = +1 (inverse, unnormalised) or -1 (forward).  N in {2,3,4,6,8,12,16}; composite sizes are one
// Cooley-Tukey split A x B done with compile-time indices, so after full unrolling everything is
// register renaming plus FADD/FMUL/FFMA with immediate twiddles (no local memory, no tables).
#pragma once
#include <cuda_runtime.h>

#include <cmath>

#ifndef GX_HD
#define GX_HD __host__ __device__ __forceinline__     // tests/host_emul runs the same functions on the CPU
#endif

namespace gx {

GX_HD float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
GX_HD float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
GX_HD float2 cmul(float2 a, float2 b) {
    return make_float2(fmaf(-a.y, b.y, a.x * b.x), fmaf(a.y, b.x, a.x * b.y));
}
GX_HD float2 cmul_conj(float2 a, float2 b) {   // a * conj(b)
    return make_float2(fmaf(a.y, b.y, a.x * b.x), fmaf(a.y, b.x, -a.x * b.y));
}
// multiply by S*i
template <int S> GX_HD float2 mul_i(float2 a) {
    return S > 0 ? make_float2(-a.y, a.x) : make_float2(a.y, -a.x);
}

// cos(2 pi t / 192), t = 0..191, from a quarter-wave table of fp64 values (rounded to fp32 at use).
// 192 = lcm(48, 64): covers every twiddle of the radices 2..16 (N | 48) and of the 32- and 64-point
// single-thread transforms.
__host__ __device__ constexpr double cos192(int t) {
    constexpr double C[49] = {
        1.00000000000000000000, 0.99946458747636568454, 0.99785892323860347908, 0.99518472667219692873,
        0.99144486137381038215, 0.98664333208487897675, 0.98078528040323043058, 0.97387697927733363201,
        0.96592582628906831221, 0.95694033573220882438, 0.94693012949510568799, 0.93590592675732575678,
        0.92387953251128673848, 0.91086382492117579091, 0.89687274153268836674, 0.88192126434835504956,
        0.86602540378443870761, 0.84920218152657889199, 0.83146961230254523567, 0.81284668459161524279,
        0.79335334029123516508, 0.77301045336273699338, 0.75183980747897738439, 0.72986407269783570850,
        0.70710678118654757274, 0.68359230202287124545, 0.65934581510006884386, 0.63439328416364548779,
        0.60876142900872065589, 0.58247769686780215270, 0.55557023301960239969, 0.52806785065036809801,
        0.50000000000000011102, 0.47139673682599758653, 0.44228869021900124592, 0.41270702980439472052,
        0.38268343236508983729, 0.35225004792123359998, 0.32143946530316169774, 0.29028467725446249759,
        0.25881904510252073948, 0.22707626303437344895, 0.19509032201612833135, 0.16289547339458881892,
        0.13052619222005171218, 0.09801714032956054812, 0.06540312923014326985, 0.03271908282177616450,
        0.00000000000000000000};
    t = ((t % 192) + 192) % 192;
    if (t > 96) t = 192 - t;         // cos(-a) = cos(a)
    return t <= 48 ? C[t] : -C[96 - t];
}
__host__ __device__ constexpr double sin192(int t) { return cos192(t - 48); }
__host__ __device__ constexpr double cos48(int t) { return cos192(4 * t); }
__host__ __device__ constexpr double sin48(int t) { return sin192(4 * t); }

// v *= e^{S 2 pi i t / N} with t, N compile-time after unrolling; trivial cases cost no multiply.
template <int N, int S> GX_HD float2 twiddle(float2 v, int t) {
    static_assert(192 % N == 0, "N must divide 192");
    const int a = ((t * (192 / N)) % 192 + 192) % 192;
    if (a == 0) return v;
    if (a == 48) return mul_i<S>(v);
    if (a == 96) return make_float2(-v.x, -v.y);
    if (a == 144) return mul_i<-S>(v);
    if (a % 48 == 24) {               // (+-1 +- i)/sqrt(2): two adds, two multiplies
        const float h = 0.70710678118654752440f;
        const float cr = (a == 24 || a == 168) ? h : -h;
        const float ci = ((a == 24 || a == 72) ? h : -h) * (S > 0 ? 1.f : -1.f);
        const float p = v.x * h, q = v.y * h;
        const float sr = cr > 0 ? 1.f : -1.f, si = ci > 0 ? 1.f : -1.f;
        return make_float2(sr * p - si * q, si * p + sr * q);
    }
    const float c = (float)cos192(a);
    const float s = (float)sin192(a) * (S > 0 ? 1.f : -1.f);
    return make_float2(fmaf(-v.y, s, v.x * c), fmaf(v.x, s, v.y * c));
}

// ZM: bit n set <=> input v[n] is known to be zero at compile time (2/3-rule padding).  The IEEE rules
// forbid the compiler from folding x + 0 (sign of zero), so the base cases skip those adds explicitly;
// a size that ignores ZM is still correct because the masked inputs really hold 0.
typedef unsigned long long zm_t;
template <int N, int S, zm_t ZM = 0ull> struct Dft;

GX_HD float2 cneg(float2 a) { return make_float2(-a.x, -a.y); }

template <int S, zm_t ZM> struct Dft<2, S, ZM> {
    GX_HD static void run(float2 (&v)[2]) {
        constexpr bool z0 = ZM & 1u, z1 = ZM & 2u;
        const float2 a = v[0], b = v[1];
        if constexpr (z1) { v[1] = a; }                       // (a, a); also covers both zero
        else if constexpr (z0) { v[0] = b; v[1] = cneg(b); }
        else { v[0] = cadd(a, b); v[1] = csub(a, b); }
    }
};

template <int S, zm_t ZM> struct Dft<3, S, ZM> {
    GX_HD static void run(float2 (&v)[3]) {
        const float2 t = cadd(v[1], v[2]);
        const float2 d = csub(v[1], v[2]);
        const float2 m = make_float2(fmaf(-0.5f, t.x, v[0].x), fmaf(-0.5f, t.y, v[0].y));
        const float h = 0.86602540378443864676f;
        const float2 r = mul_i<S>(make_float2(h * d.x, h * d.y));
        v[0] = cadd(v[0], t);
        v[1] = cadd(m, r);
        v[2] = csub(m, r);
    }
};

template <int S, zm_t ZM> struct Dft<4, S, ZM> {
    GX_HD static void run(float2 (&v)[4]) {
        constexpr bool z0 = ZM & 1u, z1 = ZM & 2u, z2 = ZM & 4u, z3 = ZM & 8u;
        float2 a, b, c, d;                                    // a = v0+v2, b = v0-v2, c = v1+v3, d = v1-v3
        if constexpr (z2) { a = v[0]; b = v[0]; }
        else if constexpr (z0) { a = v[2]; b = cneg(v[2]); }
        else { a = cadd(v[0], v[2]); b = csub(v[0], v[2]); }
        if constexpr (z3) { c = v[1]; d = v[1]; }
        else if constexpr (z1) { c = v[3]; d = cneg(v[3]); }
        else { c = cadd(v[1], v[3]); d = csub(v[1], v[3]); }
        d = mul_i<S>(d);
        if constexpr (z1 && z3) { v[0] = a; v[1] = b; v[2] = a; v[3] = b; }
        else if constexpr (z0 && z2) { v[0] = c; v[1] = d; v[2] = cneg(c); v[3] = cneg(d); }
        else { v[0] = cadd(a, c); v[1] = cadd(b, d); v[2] = csub(a, c); v[3] = csub(b, d); }
    }
};

// One Cooley-Tukey split N = A*B:  n = n1*B + n2,  k = k1 + A*k2.
template <int A, int B, zm_t ZM, int n2> __host__ __device__ constexpr zm_t sub_mask_first() {
    zm_t m = 0;
    for (int n1 = 0; n1 < A; ++n1)
        if (ZM & (1ull << (n1 * B + n2))) m |= 1ull << n1;
    return m;
}
template <int A, int B, zm_t ZM> __host__ __device__ constexpr zm_t sub_mask_second() {   // column n2 entirely zero
    zm_t m = 0;
    for (int n2 = 0; n2 < B; ++n2) {
        bool all = true;
        for (int n1 = 0; n1 < A; ++n1)
            if (!(ZM & (1ull << (n1 * B + n2)))) all = false;
        if (all) m |= 1ull << n2;
    }
    return m;
}

template <int N, int A, int B, int S, zm_t ZM, int n2>
GX_HD void dft_split_col(const float2 (&v)[N], float2 (&y)[N]) {
    float2 t[A];
#pragma unroll
    for (int n1 = 0; n1 < A; ++n1) t[n1] = v[n1 * B + n2];
    Dft<A, S, sub_mask_first<A, B, ZM, n2>()>::run(t);
#pragma unroll
    for (int k1 = 0; k1 < A; ++k1) y[k1 * B + n2] = twiddle<N, S>(t[k1], n2 * k1);
    if constexpr (n2 + 1 < B) dft_split_col<N, A, B, S, ZM, n2 + 1>(v, y);
}

template <int N, int A, int B, int S, zm_t ZM = 0ull> GX_HD void dft_split(float2 (&v)[N]) {
    static_assert(A * B == N, "bad split");
    float2 y[N];
    dft_split_col<N, A, B, S, ZM, 0>(v, y);
#pragma unroll
    for (int k1 = 0; k1 < A; ++k1) {
        float2 u[B];
#pragma unroll
        for (int n2 = 0; n2 < B; ++n2) u[n2] = y[k1 * B + n2];
        Dft<B, S, sub_mask_second<A, B, ZM>()>::run(u);
#pragma unroll
        for (int k2 = 0; k2 < B; ++k2) v[k1 + A * k2] = u[k2];
    }
}

template <int S, zm_t ZM> struct Dft<6, S, ZM> {
    GX_HD static void run(float2 (&v)[6]) { dft_split<6, 2, 3, S, ZM>(v); }
};
template <int S, zm_t ZM> struct Dft<8, S, ZM> {
    GX_HD static void run(float2 (&v)[8]) { dft_split<8, 2, 4, S, ZM>(v); }
};
template <int S, zm_t ZM> struct Dft<12, S, ZM> {
    GX_HD static void run(float2 (&v)[12]) { dft_split<12, 3, 4, S, ZM>(v); }
};
template <int S, zm_t ZM> struct Dft<16, S, ZM> {
    GX_HD static void run(float2 (&v)[16]) { dft_split<16, 4, 4, S, ZM>(v); }
};

template <int S, zm_t ZM> struct Dft<32, S, ZM> {
    GX_HD static void run(float2 (&v)[32]) { dft_split<32, 4, 8, S, ZM>(v); }
};
template <int S, zm_t ZM> struct Dft<64, S, ZM> {
    GX_HD static void run(float2 (&v)[64]) { dft_split<64, 8, 8, S, ZM>(v); }
};

template <int N, int S, zm_t ZM = 0ull> GX_HD void dft(float2 (&v)[N]) { Dft<N, S, ZM>::run(v); }

}  // namespace gx
