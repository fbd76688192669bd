// nl_pair_kernels.cuh -- packed-FP32 (FADD2/FMUL2/FFMA2) kernels of the nonlinear E×B term, sm_100a.
// PAPER.md lines 646-655 (App. D Eq. D1 line 1, zero padding); rows a1-a7 of SURVEY.md section 8(a).
//
// Same dataflow as nl_kernels.cuh (one CTA owns one (kx,ky) plane from compact spectral input to compact
// spectral output; digit-permuted real space; complex packing of the two derivative fields on the way
// in and of two real rows on the way out; zero columns never transformed), but every thread carries TWO
// independent 1D transforms through the packed FP32 instructions (dft_pairs.cuh):
//   x passes:  lane a / lane b = two ky columns  (2t, 2t+1)  resp.  (-2t, -(2t+1))
//   y passes:  lane a / lane b = two x rows      (r, r + NX/2)
// Shared-memory layouts (all fp32 words):
//   Fq   [kx row i][ky pair t] quads (re_2t, re_2t+1, im_2t, im_2t+1)         compact spectrum after a2
//   W    planar: Wre[row*RS + slot], Wim[..]; slot(q>=0) = (q&1 ? NPAIR : 0) + q/2,
//        slot(q<0) = (|q|&1 ? NPAIR : 0) + NP + |q|/2; RS = 2*NAKY + 1 is odd, so the 32-bit accesses of
//        the x passes (lanes over column pairs) and of the y passes (lanes over rows) are conflict-free.
//        The column "-0" (lane a of pair NP) is a dummy: it is transformed but never read.
//   S    [y position][row pair] quads (re_a, re_b, im_a, im_b)                 one batch of RB rows
//   W2   (forward) planar in the W region, slot2(k) = (k&1 ? NP : 0) + k/2, k = 0..Q
// Row quadruple of item rq (r0 = bt*RB/4 + rq < NX/4): h=0: rows (r0, r0+NX/2), h=1: rows (r0+NX/4,
// r0+3NX/4); the forward transform packs h=0 as real and h=1 as imaginary part.
// Real-space chi planes (workspace dchi): quads (-d_x chi(r), -d_x chi(r+NX/2), d_y chi(r), d_y chi(r+NX/2))
// at [y position][r], r < NX/2.
#pragma once
#include <type_traits>

#include "dft_pairs.cuh"
#include "nl_kernels.cuh"

namespace gx {

template <int NX_, int NY_, int RX1_, int RX2_, int RY1_, int RY2_, int RB_, int NT_, int MINB_>
struct PairCfg {
    static constexpr int NX = NX_, NY = NY_, RX1 = RX1_, RX2 = RX2_, RY1 = RY1_, RY2 = RY2_;
    static constexpr int RB = RB_, NT = NT_, MINB = MINB_;
    static constexpr int K = (NX - 1) / 3, Q = (NY - 1) / 3;
    static constexpr int NAKX = 2 * K + 1, NAKY = Q + 1, NK = NAKX * NAKY;
    static constexpr int NP = NAKY / 2, NPAIR = 2 * NP, NSLOT = 2 * NPAIR, RS = NSLOT + 1;
    static constexpr int QB = RB / 4, HB = RB / 2, NBATCH = NX / RB;
    static constexpr int W_WORDS = ((2 * NX * RS + 3) / 4) * 4;           // two planes, 16-byte multiple
    static constexpr int S_WORDS_MIN = NY * HB * 4;
    static constexpr int S_WORDS = (2 * NK > S_WORDS_MIN) ? 2 * NK : S_WORDS_MIN;
    static constexpr int SMEM_BYTES = (W_WORDS + S_WORDS) * 4 + (NX + NY) * 8;
    static constexpr unsigned zero_mask(int R1, int R2, int N, int KK) {
        unsigned m = 0;
        for (int n1 = 0; n1 < R1; ++n1)
            if (!(n1 * R2 <= KK || n1 * R2 + R2 - 1 >= N - KK)) m |= 1u << n1;
        return m;
    }
    static constexpr unsigned ZMX = zero_mask(RX1, RX2, NX, K), ZMY = zero_mask(RY1, RY2, NY, Q);
    static_assert(RX1 * RX2 == NX && RY1 * RY2 == NY, "radix split");
    static_assert(NAKY % 2 == 0, "column pairs need an even number of kept ky");
    static_assert(NX % 4 == 0 && RB % 4 == 0 && NX % RB == 0, "row quadruples");
    static_assert(RY2 % 2 == 0 && NY % 2 == 0, "slot arithmetic assumes even RY2, NY");
    static_assert(SMEM_BYTES <= 232448, "plane does not fit in shared memory");
};

// ------------------------------------------------------------------------------------------------
// inverse x transform of U(k) = (i kx - ky) f(k); Fq in shared memory, result in the planar W.
template <class C>
__device__ __forceinline__ void px_inverse(float* __restrict__ W, const float2* __restrict__ twx,
                                           float dkx, float dky, const float4* __restrict__ Fq) {
    constexpr int NX = C::NX, K = C::K, NAKX = C::NAKX, NP = C::NP, NPAIR = C::NPAIR, RS = C::RS;
    constexpr int R1 = C::RX1, R2 = C::RX2, IM = NX * RS;
    for (int t = threadIdx.x; t < R2 * NPAIR; t += C::NT) {
        const int n2 = t / NPAIR, p = t - n2 * NPAIR;
        const bool neg = p >= NP;                          // columns q <= 0
        const int tp = neg ? p - NP : p;                   // |q| = 2 tp, 2 tp + 1
        const float sgn = neg ? -1.f : 1.f;                // q < 0: f(a,q) = conj f(-a,-q)
        const float kya = dky * (float)(2 * tp), kyb = dky * (float)(2 * tp + 1);
        const u64 nky = pk2(-sgn * kya, -sgn * kyb);       // -ky per lane
        const u64 snky = pk2(-kya, -kyb);                  // sgn * (-ky)
        const int stepP = neg ? -R2 * NP : R2 * NP;
        const float4* __restrict__ FP = Fq + (neg ? (NAKX - n2) * NP : n2 * NP) + tp;
        const float4* __restrict__ FN = Fq + (neg ? (NX - n2) * NP : (n2 - NX + NAKX) * NP) + tp;
        const float an2 = (float)n2, an2n = (float)(n2 - NX);
        c2 v[R1];
#pragma unroll
        for (int n1 = 0; n1 < R1; ++n1) {
            const int lo = n1 * R2, hi = n1 * R2 + R2 - 1;
            const bool allP = hi <= K, someP = lo <= K;
            const bool allN = lo >= NX - K, someN = hi >= NX - K;
            v[n1] = czero2();
            if (someP || someN) {
                float4 f = make_float4(0.f, 0.f, 0.f, 0.f);
                float kxa = 0.f;
                if (someP) {
                    const bool isP = allP || (lo + n2 <= K);
                    const float4* ptr = FP + n1 * stepP;
                    if (n1 == 0 && neg && n2 == 0) ptr = Fq + tp;     // mode a = 0: -a is row 0
                    if (isP) { f = *ptr; kxa = dkx * (an2 + (float)lo); }
                }
                if (someN) {
                    const bool isN = allN || (lo + n2 >= NX - K);
                    if (isN) { f = *(FN + n1 * stepP); kxa = dkx * (an2n + (float)lo); }
                }
                const u64 fx = pk2(f.x, f.y), fi = pk2(f.z, f.w);
                // U = (-ky fx - kx fy, kx fx - ky fy), fy = sgn * fi
                v[n1].re = fma2(fx, nky, mul2(fi, bc2(-sgn * kxa)));
                v[n1].im = fma2(fx, bc2(kxa), mul2(fi, snky));
            }
        }
        dft2<R1, +1, C::ZMX>(v);
        float* __restrict__ Wa = W + n2 * RS + p;
#pragma unroll
        for (int k1 = 0; k1 < R1; ++k1) {
            c2 o = v[k1];
            if (k1 != 0) { const float2 w = twx[n2 * k1]; o = cmul_s(o, w.x, w.y); }
            float ra, rb, ia, ib;
            upk2(o.re, ra, rb); upk2(o.im, ia, ib);
            float* d = Wa + k1 * R2 * RS;
            d[0] = ra; d[NPAIR] = rb; d[IM] = ia; d[IM + NPAIR] = ib;
        }
    }
    __syncthreads();
    GX_PHASE(22);
    for (int t = threadIdx.x; t < R1 * NPAIR; t += C::NT) {
        const int k1 = t / NPAIR, p = t - k1 * NPAIR;
        float* __restrict__ Wa = W + k1 * R2 * RS + p;
        c2 v[R2];
#pragma unroll
        for (int n2 = 0; n2 < R2; ++n2) {
            const float* s = Wa + n2 * RS;
            v[n2].re = pk2(s[0], s[NPAIR]); v[n2].im = pk2(s[IM], s[IM + NPAIR]);
        }
        dft2<R2, +1>(v);
#pragma unroll
        for (int k2 = 0; k2 < R2; ++k2) {
            float ra, rb, ia, ib;
            upk2(v[k2].re, ra, rb); upk2(v[k2].im, ia, ib);
            float* d = Wa + k2 * RS;
            d[0] = ra; d[NPAIR] = rb; d[IM] = ia; d[IM + NPAIR] = ib;
        }
    }
    __syncthreads();
}

// y inverse pass 1 for one batch: planar W (non-zero columns) -> S[(k1*RY2+n2)*HB + rp] quads.
// rp = h*QB + rq: rows (ra, ra + NX/2), ra = h*NX/4 + bt*QB + rq.
template <class C>
__device__ __forceinline__ void py_inverse_pass1(const float* __restrict__ W, float4* __restrict__ S,
                                                 const float2* __restrict__ twy, int bt) {
    constexpr int NX = C::NX, NY = C::NY, Q = C::Q, NP = C::NP, NPAIR = C::NPAIR, RS = C::RS;
    constexpr int R1 = C::RY1, R2 = C::RY2, HB = C::HB, QB = C::QB, IM = NX * RS, RBO = (NX / 2) * RS;
    for (int t = threadIdx.x; t < R2 * HB; t += C::NT) {
        const int n2 = t / HB, rp = t - n2 * HB;
        const int h = rp / QB, rq = rp - h * QB;
        const int ra = h * (NX / 4) + bt * QB + rq;
        const int odd = n2 & 1;
        // column q = lo + n2 >= 0:  slot = (odd ? NPAIR : 0) + lo/2 + n2/2
        // column q = lo + n2 - NY < 0: |q| = NY - lo - n2, slot = (odd ? NPAIR : 0) + NP + (NY - lo)/2 - (n2+1)/2
        const float* __restrict__ WP = W + ra * RS + (odd ? NPAIR : 0) + n2 / 2;
        const float* __restrict__ WN = W + ra * RS + (odd ? NPAIR : 0) + NP + NY / 2 - (n2 + 1) / 2;
        c2 v[R1];
#pragma unroll
        for (int n1 = 0; n1 < R1; ++n1) {
            const int lo = n1 * R2, hi = n1 * R2 + R2 - 1;
            const bool allP = hi <= Q, someP = lo <= Q, allN = lo >= NY - Q, someN = hi >= NY - Q;
            v[n1] = czero2();
            if (someP && (allP || lo + n2 <= Q)) {
                const float* s = WP + lo / 2;
                v[n1].re = pk2(s[0], s[RBO]); v[n1].im = pk2(s[IM], s[IM + RBO]);
            }
            if (someN && (allN || lo + n2 >= NY - Q)) {
                const float* s = WN - lo / 2;
                v[n1].re = pk2(s[0], s[RBO]); v[n1].im = pk2(s[IM], s[IM + RBO]);
            }
        }
        dft2<R1, +1, C::ZMY>(v);
#pragma unroll
        for (int k1 = 0; k1 < R1; ++k1) {
            c2 o = v[k1];
            if (k1 != 0) { const float2 w = twy[n2 * k1]; o = cmul_s(o, w.x, w.y); }
            float ra_, rb_, ia_, ib_;
            upk2(o.re, ra_, rb_); upk2(o.im, ia_, ib_);
            S[(k1 * R2 + n2) * HB + rp] = make_float4(ra_, rb_, ia_, ib_);
        }
    }
    __syncthreads();
}

__device__ __forceinline__ c2 ld_quad(const float4* p) {
    const float4 f = *p;
    c2 r; r.re = pk2(f.x, f.y); r.im = pk2(f.z, f.w);
    return r;
}
__device__ __forceinline__ void st_quad(float4* p, c2 v) {
    float a, b, c, d;
    upk2(v.re, a, b); upk2(v.im, c, d);
    *p = make_float4(a, b, c, d);
}

// forward x transform on the kept columns (pairs (2t, 2t+1)); planar W2 -> compact out (times scale)
template <class C>
__device__ __forceinline__ void px_forward(float* __restrict__ W, const float2* __restrict__ twx,
                                           float2* __restrict__ out, float scale) {
    constexpr int NX = C::NX, K = C::K, NAKX = C::NAKX, NAKY = C::NAKY, NP = C::NP, RS = C::RS;
    constexpr int R1 = C::RX1, R2 = C::RX2, IM = NX * RS;
    for (int t = threadIdx.x; t < R1 * NP; t += C::NT) {
        const int a = t / NP, tp = t - a * NP;
        float* __restrict__ Wa = W + a * R2 * RS + tp;
        c2 v[R2];
#pragma unroll
        for (int b = 0; b < R2; ++b) {
            const float* s = Wa + b * RS;
            v[b].re = pk2(s[0], s[NP]); v[b].im = pk2(s[IM], s[IM + NP]);
        }
        dft2<R2, -1>(v);
#pragma unroll
        for (int d = 0; d < R2; ++d) {
            c2 o = v[d];
            if (d != 0) { const float2 w = twx[a * d]; o = cmul_s(o, w.x, -w.y); }
            float ra, rb, ia, ib;
            upk2(o.re, ra, rb); upk2(o.im, ia, ib);
            float* dst = Wa + d * RS;
            dst[0] = ra; dst[NP] = rb; dst[IM] = ia; dst[IM + NP] = ib;
        }
    }
    __syncthreads();
    GX_PHASE(23);
    for (int t = threadIdx.x; t < R2 * NP; t += C::NT) {
        const int d = t / NP, tp = t - d * NP;
        const float* __restrict__ Wa = W + d * RS + tp;
        c2 v[R1];
#pragma unroll
        for (int a = 0; a < R1; ++a) {
            const float* s = Wa + a * R2 * RS;
            v[a].re = pk2(s[0], s[NP]); v[a].im = pk2(s[IM], s[IM + NP]);
        }
        dft2<R1, -1>(v);
        const u64 sc = bc2(scale);
#pragma unroll
        for (int cc = 0; cc < R1; ++cc) {
            if (cc * R2 <= K || cc * R2 + R2 - 1 >= NX - K) {
                const int n = d + R2 * cc;
                int i = -1;
                if (n <= K) i = n;
                else if (n >= NX - K) i = n - NX + NAKX;
                if (i >= 0) {
                    float ra, rb, ia, ib;
                    upk2(mul2(v[cc].re, sc), ra, rb); upk2(mul2(v[cc].im, sc), ia, ib);
                    *reinterpret_cast<float4*>(out + i * NAKY + 2 * tp) = make_float4(ra, ia, rb, ib);
                }
            }
        }
    }
}

// raw planes staged by TMA -> Laguerre row combine in registers -> Fq quads in the S region
template <class C>
__device__ __forceinline__ void pstage_combine_tma(float* __restrict__ raw, float4* __restrict__ Fq,
                                                   unsigned long long* bar, unsigned& parity,
                                                   const float2* __restrict__ planes, size_t lstride,
                                                   const float* __restrict__ coef, int Nl) {
    constexpr int NK = C::NK, NT = C::NT, NK2 = NK / 2;
    constexpr int CAP = (C::W_WORDS + C::S_WORDS) / (2 * NK);
    constexpr int PER = (NK2 + NT - 1) / NT;
    static_assert(CAP >= 1, "TMA staging needs room for one plane");
    const float4* __restrict__ raw4 = reinterpret_cast<const float4*>(raw) + threadIdx.x;
    float4 acc[PER];
#pragma unroll
    for (int u = 0; u < PER; ++u) acc[u] = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int l0 = 0; l0 < Nl; l0 += CAP) {
        const int nl = min(CAP, Nl - l0);
        if (threadIdx.x == 0) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            mbar_expect_tx(bar, (unsigned)(nl * NK * sizeof(float2)));
            for (int l = 0; l < nl; ++l)
                bulk_g2s(raw + (size_t)l * 2 * NK, planes + (size_t)(l0 + l) * lstride, NK * sizeof(float2), bar);
        }
        mbar_wait(bar, parity);
        parity ^= 1u;
        for (int l = 0; l < nl; ++l) {
            const float t = coef[l0 + l];
            const float4* __restrict__ src = raw4 + l * NK2;
#pragma unroll
            for (int u = 0; u < PER; ++u) {
                if ((u + 1) * NT <= NK2 || (int)threadIdx.x + u * NT < NK2) {
                    const float4 f = src[u * NT];
                    acc[u].x = fmaf(t, f.x, acc[u].x);
                    acc[u].y = fmaf(t, f.y, acc[u].y);
                    acc[u].z = fmaf(t, f.z, acc[u].z);
                    acc[u].w = fmaf(t, f.w, acc[u].w);
                }
            }
        }
        __syncthreads();                                         // raw region consumed
    }
    float4* __restrict__ F4 = Fq + threadIdx.x;
#pragma unroll
    for (int u = 0; u < PER; ++u)
        if ((u + 1) * NT <= NK2 || (int)threadIdx.x + u * NT < NK2)
            F4[u * NT] = make_float4(acc[u].x, acc[u].z, acc[u].y, acc[u].w);   // (re0, re1, im0, im1)
}

// ================================================================================================
// a1 + a3 + a4 for the potential: real-space chi quads of chi_{s,z,j} = M_{s,z,j} Phi_z.
template <class C>
__global__ void __launch_bounds__(C::NT, C::MINB) chi_planes_pair_kernel(const NlParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float* W = reinterpret_cast<float*>(smem_raw);
    float4* S = reinterpret_cast<float4*>(W + C::W_WORDS);
    float2* twx = reinterpret_cast<float2*>(W + C::W_WORDS + C::S_WORDS);
    float2* twy = twx + C::NX;
    constexpr int NK2 = C::NK / 2, R1 = C::RY1, R2 = C::RY2, HB = C::HB, QB = C::QB;
    const int unit = blockIdx.x;                 // (s*Nz + z)*J + j
    const int z = (unit / p.J) % p.Nz;
    const float4* __restrict__ phi = reinterpret_cast<const float4*>(p.phi + (size_t)z * C::NK);
    const float2* __restrict__ M = reinterpret_cast<const float2*>(p.M + (size_t)unit * C::NK);
    pdl_launch_dependents();        // the bracket kernel's prologue (a2-a4 x part) does not read dchi
    load_twiddles<C>(twx, twy, p);
    for (int i = threadIdx.x; i < NK2; i += C::NT) {
        const float4 f = __ldg(phi + i);
        const float2 m = __ldg(M + i);
        S[i] = make_float4(f.x * m.x, f.z * m.y, f.y * m.x, f.w * m.y);
    }
    __syncthreads();
    px_inverse<C>(W, twx, p.dkx, p.dky, S);
    float4* __restrict__ dchi = reinterpret_cast<float4*>(p.dchi) + (size_t)unit * (C::NX / 2) * C::NY;
    for (int bt = 0; bt < C::NBATCH; ++bt) {
        py_inverse_pass1<C>(W, S, twy, bt);
        for (int t = threadIdx.x; t < R1 * HB; t += C::NT) {
            const int k1 = t / HB, rp = t - k1 * HB;
            const int h = rp / QB, rq = rp - h * QB;
            const int ra = h * (C::NX / 4) + bt * QB + rq;
            c2 v[R2];
#pragma unroll
            for (int n2 = 0; n2 < R2; ++n2) v[n2] = ld_quad(S + (k1 * R2 + n2) * HB + rp);
            dft2<R2, +1>(v);
#pragma unroll
            for (int k2 = 0; k2 < R2; ++k2) {
                c2 o; o.re = neg2(v[k2].re); o.im = v[k2].im;      // (-d_x chi, d_y chi)
                st_quad(dchi + (size_t)(k1 * R2 + k2) * (C::NX / 2) + ra, o);
            }
        }
        __syncthreads();
    }
}

// ================================================================================================
// a2-a7 for one (s,m,z,j): Bhat_j(k) = F_k[ d_y chi d_x gt - d_x chi d_y gt ], 2/3-rule truncated.
template <class C>
__global__ void __launch_bounds__(C::NT, C::MINB) bracket_pair_kernel(const NlParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float* W = reinterpret_cast<float*>(smem_raw);
    float4* S = reinterpret_cast<float4*>(W + C::W_WORDS);
    float2* twx = reinterpret_cast<float2*>(W + C::W_WORDS + C::S_WORDS);
    float2* twy = twx + C::NX;
    constexpr int NX = C::NX, NY = C::NY, Q = C::Q, NK = C::NK, NP = C::NP, RS = C::RS;
    constexpr int R1 = C::RY1, R2 = C::RY2, HB = C::HB, QB = C::QB, IM = NX * RS;

    const int unit = blockIdx.x;                 // ((s*Nz + z)*J + j)*Nm + m
    const int m = unit % p.Nm;
    const int szj = unit / p.Nm;
    const int j = szj % p.J;
    const int z = (szj / p.J) % p.Nz;
    const int s = szj / (p.J * p.Nz);
    const size_t lstride = (size_t)p.Nz * NK;
    const float2* __restrict__ g0 = p.g + ((size_t)(s * p.Nm + m) * p.Nl * p.Nz + z) * NK;

    __shared__ unsigned long long stage_bar;
    __shared__ float Tsh[16];
    unsigned bar_parity = 0;
    GX_PHASE(0);
    if (threadIdx.x == 0) mbar_init(&stage_bar, 1);
    if (threadIdx.x < p.Nl) Tsh[threadIdx.x] = __ldg(p.T + j * p.Nl + threadIdx.x);
    __syncthreads();
    pdl_launch_dependents();
    load_twiddles<C>(twx, twy, p);
    // ---- a2: forward Laguerre transform l -> node j, fused into the load
    pstage_combine_tma<C>(W, S, &stage_bar, bar_parity, g0, lstride, Tsh, p.Nl);
    __syncthreads();
    GX_PHASE(1);
    // ---- a3 + a4 (x part)
    px_inverse<C>(W, twx, p.dkx, p.dky, S);
    GX_PHASE(2);

    const float4* __restrict__ dchi = reinterpret_cast<const float4*>(p.dchi) + (size_t)szj * (NX / 2) * NY;
    pdl_wait();                     // chi planes of this call are complete and visible from here on
    for (int bt = 0; bt < C::NBATCH; ++bt) {
        // ---- a4 (y part, first pass)
        GX_PHASE(3 + 3 * bt);
        py_inverse_pass1<C>(W, S, twy, bt);
        GX_PHASE(4 + 3 * bt);
        // ---- a4 (last pass) + a5 bracket + a6 (first forward pass), all in registers
        for (int t = threadIdx.x; t < R1 * QB; t += C::NT) {
            const int k1 = t / QB, rq = t - k1 * QB;
            c2 c[R2];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int ra = h * (NX / 4) + bt * QB + rq;
                c2 v[R2];
#pragma unroll
                for (int n2 = 0; n2 < R2; ++n2) v[n2] = ld_quad(S + (k1 * R2 + n2) * HB + h * QB + rq);
                dft2<R2, +1>(v);
#pragma unroll
                for (int k2 = 0; k2 < R2; ++k2) {
                    const float4 d = __ldg(dchi + (size_t)(k1 * R2 + k2) * (NX / 2) + ra);
                    // d_y chi d_x g - d_x chi d_y g  (d.x, d.y hold -d_x chi)
                    const u64 b = fma2(pk2(d.z, d.w), v[k2].re, mul2(pk2(d.x, d.y), v[k2].im));
                    if (h == 0) c[k2].re = b; else c[k2].im = b;
                }
            }
            dft2<R2, -1>(c);
#pragma unroll
            for (int d = 0; d < R2; ++d) {
                c2 o = c[d];
                if (d != 0) { const float2 w = twy[k1 * d]; o = cmul_s(o, w.x, -w.y); }
                st_quad(S + (k1 * R2 + d) * HB + rq, o);
            }
        }
        __syncthreads();
        GX_PHASE(5 + 3 * bt);
        // ---- a6 (last y pass) + a7 (keep ky <= Q) + separation of the packed rows
        for (int t = threadIdx.x; t < (R2 / 2 + 1) * QB; t += C::NT) {
            const int dd = t / QB, rq = t - dd * QB;
            const int d0 = dd, d1 = (R2 - dd) % R2;
            c2 u0[R1], u1[R1];
#pragma unroll
            for (int a = 0; a < R1; ++a) u0[a] = ld_quad(S + (a * R2 + d0) * HB + rq);
            dft2<R1, -1>(u0);
            if (d1 != d0) {
#pragma unroll
                for (int a = 0; a < R1; ++a) u1[a] = ld_quad(S + (a * R2 + d1) * HB + rq);
                dft2<R1, -1>(u1);
            } else {
#pragma unroll
                for (int a = 0; a < R1; ++a) u1[a] = u0[a];
            }
            // rows: W0 -> (r0, r0+NX/2), W1 -> (r0+NX/4, r0+3NX/4), r0 = bt*QB + rq
            float* __restrict__ W0 = W + (bt * QB + rq) * RS;
            const u64 half = bc2(0.5f);
            auto emit = [&](int k, c2 A, c2 B) {
                // Zre = (A + conj B)/2,  Zim = (A - conj B)/(2i)
                const u64 r0 = mul2(add2(A.re, B.re), half), i0 = mul2(sub2(A.im, B.im), half);
                const u64 r1 = mul2(add2(A.im, B.im), half), i1 = mul2(sub2(B.re, A.re), half);
                float* d = W0 + ((k & 1) ? NP : 0) + (k >> 1);
                float xa, xb;
                upk2(r0, xa, xb); d[0] = xa; d[(NX / 2) * RS] = xb;
                upk2(i0, xa, xb); d[IM] = xa; d[IM + (NX / 2) * RS] = xb;
                upk2(r1, xa, xb); d[(NX / 4) * RS] = xa; d[(3 * NX / 4) * RS] = xb;
                upk2(i1, xa, xb); d[IM + (NX / 4) * RS] = xa; d[IM + (3 * NX / 4) * RS] = xb;
            };
#pragma unroll
            for (int cc = 0; cc <= Q / R2; ++cc) {
                {
                    const int k = d0 + R2 * cc;
                    if (k <= Q) emit(k, u0[cc], (d0 == 0) ? u1[(R1 - cc) % R1] : u1[R1 - 1 - cc]);
                }
                if (d1 != d0) {
                    const int k = d1 + R2 * cc;
                    if (k <= Q) emit(k, u1[cc], u0[R1 - 1 - cc]);
                }
            }
        }
        __syncthreads();
    }
    // ---- a6 (x part) + a7 (keep |kx| <= K)
    GX_PHASE(20);
    px_forward<C>(W, twx, p.bhat + (size_t)unit * NK, p.scale);

    // ---- publish: CTA barrier orders every thread's stores before thread 0's gpu-scope fence (cumulative)
    __syncthreads();
    GX_PHASE(21);
    if (threadIdx.x == 0) { __threadfence(); atomicAdd(p.count + (s * p.Nm + m) * p.Nz + z, 1u); }
}

// ================================================================================================
// Persistent, warp-asynchronous variant of bracket_pair_kernel (profiles/r01b_*: the block-synchronous
// kernel spends most of its time at CTA barriers and in partially filled passes).  One CTA per SM loops
// over units; inside a unit only three CTA barriers remain (columns -> rows -> columns -> next unit):
//   x inverse : warp w owns ky pair groups tp = w, w+NW, ... (columns (2tp,2tp+1) and their mirror
//               images); both x passes of a group are warp-local (__syncwarp).  The Laguerre row
//               combine (a2) is done on the fly from the TMA-staged raw planes.
//   y part    : warp w owns groups of 4 row quadruples; y pass 1, the fused bracket pass and the last
//               forward y pass run through a private 8-row-pair tile with an XOR swizzle.
//   x forward : warp w owns kept ky pairs tp = w, w+NW, ...
// The raw planes of the NEXT unit are fetched by TMA into the (then idle) tile region while the x
// forward passes of the current unit run.
template <int NX_, int NY_, int RX1_, int RX2_, int RY1_, int RY2_, int NW_, int MAXL_>
struct PersistCfg {
    static constexpr int NX = NX_, NY = NY_, RX1 = RX1_, RX2 = RX2_, RY1 = RY1_, RY2 = RY2_;
    static constexpr int NW = NW_, NT = 32 * NW_, MAXL = MAXL_;
    static constexpr int K = (NX - 1) / 3, Q = (NY - 1) / 3;
    static constexpr int NAKX = 2 * K + 1, NAKY = Q + 1, NK = NAKX * NAKY;
    static constexpr int NP = NAKY / 2, NPAIR = 2 * NP, NSLOT = 2 * NPAIR, RS = NSLOT + 1;
    static constexpr int NQG = NX / 16;                                   // groups of 4 row quadruples
    static constexpr int W_WORDS = ((2 * NX * RS + 3) / 4) * 4;
    static constexpr int TILE_QUADS = NY * 8;
    static constexpr int S_WORDS_TILES = NW * TILE_QUADS * 4;
    static constexpr int RAW_WORDS = MAXL * 2 * NK;
    static constexpr int S_WORDS = S_WORDS_TILES > RAW_WORDS ? S_WORDS_TILES : RAW_WORDS;
    static constexpr int SMEM_BYTES = (W_WORDS + S_WORDS) * 4 + (NX + NY) * 8;
    static constexpr unsigned zero_mask(int R1, int R2, int N, int KK) {
        unsigned m = 0;
        for (int n1 = 0; n1 < R1; ++n1)
            if (!(n1 * R2 <= KK || n1 * R2 + R2 - 1 >= N - KK)) m |= 1u << n1;
        return m;
    }
    static constexpr unsigned ZMX = zero_mask(RX1, RX2, NX, K), ZMY = zero_mask(RY1, RY2, NY, Q);
    static_assert(RX1 * RX2 == NX && RY1 * RY2 == NY, "radix split");
    static_assert(NAKY % 2 == 0 && NK % 2 == 0, "column pairs need an even number of kept ky");
    static_assert(NX % 16 == 0, "groups of 4 row quadruples");
    static_assert(RY2 % 4 == 0 && NY % 2 == 0, "y pass 1 rounds");
    static_assert(2 * RX2 <= 32 && 2 * RX1 <= 32, "x items of one group fit one warp round");
    static_assert(SMEM_BYTES <= 232448, "does not fit in shared memory");
};

template <class C>
__global__ void __launch_bounds__(C::NT, 1) bracket_persist_kernel(const NlParams p, int nunits) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float* W = reinterpret_cast<float*>(smem_raw);
    float4* S = reinterpret_cast<float4*>(W + C::W_WORDS);
    float2* twx = reinterpret_cast<float2*>(W + C::W_WORDS + C::S_WORDS);
    float2* twy = twx + C::NX;
    constexpr int NX = C::NX, NY = C::NY, K = C::K, Q = C::Q, NK = C::NK, NAKX = C::NAKX, NAKY = C::NAKY;
    constexpr int NP = C::NP, NPAIR = C::NPAIR, RS = C::RS, IM = NX * RS, NK2 = NK / 2;
    constexpr int X1 = C::RX1, X2 = C::RX2, Y1 = C::RY1, Y2 = C::RY2;
    constexpr int RBO = (NX / 2) * RS;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float4* __restrict__ tile = S + warp * C::TILE_QUADS;
    const float4* __restrict__ raw = S;                       // [l][kx row][ky pair] quads as stored in g

    __shared__ unsigned long long full_bar;
    if (threadIdx.x == 0) mbar_init(&full_bar, 1);
    pdl_launch_dependents();
    load_twiddles<C>(twx, twy, p);
    __syncthreads();
    const size_t lstride = (size_t)p.Nz * NK;
    auto issue_load = [&](int unit) {                         // one thread
        const int m = unit % p.Nm, szj = unit / p.Nm;
        const int z = (szj / p.J) % p.Nz, s = szj / (p.J * p.Nz);
        const float2* g0 = p.g + ((size_t)(s * p.Nm + m) * p.Nl * p.Nz + z) * NK;
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        mbar_expect_tx(&full_bar, (unsigned)(p.Nl * NK * sizeof(float2)));
        for (int l = 0; l < p.Nl; ++l)
            bulk_g2s(reinterpret_cast<float*>(S) + (size_t)l * 2 * NK, g0 + (size_t)l * lstride, NK * sizeof(float2), &full_bar);
    };
    if (threadIdx.x == 0 && (int)blockIdx.x < nunits) issue_load(blockIdx.x);
    unsigned parity = 0;
    bool first = true;

    for (int unit = blockIdx.x; unit < nunits; unit += gridDim.x) {
        const int m = unit % p.Nm;
        const int szj = unit / p.Nm;
        const int j = szj % p.J;
        const int z = (szj / p.J) % p.Nz;
        const int s = szj / (p.J * p.Nz);
        float Tl[C::MAXL];
#pragma unroll
        for (int l = 0; l < C::MAXL; ++l) Tl[l] = l < p.Nl ? __ldg(p.T + j * p.Nl + l) : 0.f;
        mbar_wait(&full_bar, parity);
        parity ^= 1u;

        // ---------------- a2 + a3 + a4 (x part), warp-local per ky pair group
        for (int tp = warp; tp < NP; tp += C::NW) {
            if (lane < 2 * X2) {
                const int neg = lane >= X2;
                const int n2 = neg ? lane - X2 : lane;
                const int pcol = neg ? NP + tp : tp;
                const float sgn = neg ? -1.f : 1.f;
                const float kya = p.dky * (float)(2 * tp), kyb = p.dky * (float)(2 * tp + 1);
                const u64 nky = pk2(-sgn * kya, -sgn * kyb);
                const u64 snky = pk2(-kya, -kyb);
                const int stepP = neg ? -X2 * NP : X2 * NP;
                const float4* __restrict__ FP = raw + (neg ? (NAKX - n2) * NP : n2 * NP) + tp;
                const float4* __restrict__ FN = raw + (neg ? (NX - n2) * NP : (n2 - NX + NAKX) * NP) + tp;
                const float an2 = (float)n2, an2n = (float)(n2 - NX);
                c2 v[X1];
#pragma unroll
                for (int n1 = 0; n1 < X1; ++n1) {
                    const int lo = n1 * X2, hi = n1 * X2 + X2 - 1;
                    const bool allP = hi <= K, someP = lo <= K;
                    const bool allN = lo >= NX - K, someN = hi >= NX - K;
                    v[n1] = czero2();
                    if (someP || someN) {
                        const float4* ptr = raw;
                        bool have = false;
                        float kxa = 0.f;
                        if (someP) {
                            if (allP || (lo + n2 <= K)) {
                                ptr = FP + n1 * stepP;
                                if (n1 == 0 && neg && n2 == 0) ptr = raw + tp;
                                kxa = p.dkx * (an2 + (float)lo);
                                have = true;
                            }
                        }
                        if (someN) {
                            if (allN || (lo + n2 >= NX - K)) { ptr = FN + n1 * stepP; kxa = p.dkx * (an2n + (float)lo); have = true; }
                        }
                        if (have) {
                            // Laguerre row combine of the staged planes: f = sum_l T[j][l] G_l  (re0,im0,re1,im1)
                            u64 f01 = 0ull, f23 = 0ull;
#pragma unroll
                            for (int l = 0; l < C::MAXL; ++l) {
                                if (l < p.Nl) {
                                    const float4 g = ptr[l * NK2];
                                    f01 = fma2(pk2(g.x, g.y), bc2(Tl[l]), f01);
                                    f23 = fma2(pk2(g.z, g.w), bc2(Tl[l]), f23);
                                }
                            }
                            float re0, im0, re1, im1;
                            upk2(f01, re0, im0); upk2(f23, re1, im1);
                            const u64 fx = pk2(re0, re1), fi = pk2(im0, im1);
                            v[n1].re = fma2(fx, nky, mul2(fi, bc2(-sgn * kxa)));
                            v[n1].im = fma2(fx, bc2(kxa), mul2(fi, snky));
                        }
                    }
                }
                dft2<X1, +1, C::ZMX>(v);
                float* __restrict__ Wa = W + n2 * RS + pcol;
#pragma unroll
                for (int k1 = 0; k1 < X1; ++k1) {
                    c2 o = v[k1];
                    if (k1 != 0) { const float2 w = twx[n2 * k1]; o = cmul_s(o, w.x, w.y); }
                    float ra, rb, ia, ib;
                    upk2(o.re, ra, rb); upk2(o.im, ia, ib);
                    float* d = Wa + k1 * X2 * RS;
                    d[0] = ra; d[NPAIR] = rb; d[IM] = ia; d[IM + NPAIR] = ib;
                }
            }
            __syncwarp();
            if (lane < 2 * X1) {
                const int neg = lane >= X1;
                const int k1 = neg ? lane - X1 : lane;
                const int pcol = neg ? NP + tp : tp;
                float* __restrict__ Wa = W + k1 * X2 * RS + pcol;
                c2 v[X2];
#pragma unroll
                for (int n2 = 0; n2 < X2; ++n2) {
                    const float* sp = Wa + n2 * RS;
                    v[n2].re = pk2(sp[0], sp[NPAIR]); v[n2].im = pk2(sp[IM], sp[IM + NPAIR]);
                }
                dft2<X2, +1>(v);
#pragma unroll
                for (int k2 = 0; k2 < X2; ++k2) {
                    float ra, rb, ia, ib;
                    upk2(v[k2].re, ra, rb); upk2(v[k2].im, ia, ib);
                    float* d = Wa + k2 * RS;
                    d[0] = ra; d[NPAIR] = rb; d[IM] = ia; d[IM + NPAIR] = ib;
                }
            }
            __syncwarp();
        }
        __syncthreads();                       // A: all columns transformed, raw planes consumed

        if (first) { pdl_wait(); first = false; }      // chi planes of this call are complete from here on
        const float4* __restrict__ dchi = reinterpret_cast<const float4*>(p.dchi) + (size_t)szj * (NX / 2) * NY;
        // ---------------- a4 (y part) + a5 + a6 (y part) + a7, warp-local per group of 4 row quadruples
        for (int qg = warp; qg < C::NQG; qg += C::NW) {
            // y pass 1: lanes = (n2 = 4*rr + lane/8, rp = lane%8 = h*4 + rql)
            {
                const int rp = lane & 7, h = rp >> 2, rql = rp & 3;
                const int ra = h * (NX / 4) + 4 * qg + rql;
#pragma unroll 1
                for (int rr = 0; rr < Y2 / 4; ++rr) {
                    const int n2 = 4 * rr + (lane >> 3);
                    const int odd = n2 & 1;
                    const float* __restrict__ WP = W + ra * RS + (odd ? NPAIR : 0) + n2 / 2;
                    const float* __restrict__ WN = W + ra * RS + (odd ? NPAIR : 0) + NP + NY / 2 - (n2 + 1) / 2;
                    c2 v[Y1];
#pragma unroll
                    for (int n1 = 0; n1 < Y1; ++n1) {
                        const int lo = n1 * Y2, hi = n1 * Y2 + Y2 - 1;
                        const bool allP = hi <= Q, someP = lo <= Q, allN = lo >= NY - Q, someN = hi >= NY - Q;
                        v[n1] = czero2();
                        if (someP && (allP || lo + n2 <= Q)) {
                            const float* sp = WP + lo / 2;
                            v[n1].re = pk2(sp[0], sp[RBO]); v[n1].im = pk2(sp[IM], sp[IM + RBO]);
                        }
                        if (someN && (allN || lo + n2 >= NY - Q)) {
                            const float* sp = WN - lo / 2;
                            v[n1].re = pk2(sp[0], sp[RBO]); v[n1].im = pk2(sp[IM], sp[IM + RBO]);
                        }
                    }
                    dft2<Y1, +1, C::ZMY>(v);
#pragma unroll
                    for (int k1 = 0; k1 < Y1; ++k1) {
                        c2 o = v[k1];
                        if (k1 != 0) { const float2 w = twy[n2 * k1]; o = cmul_s(o, w.x, w.y); }
                        st_quad(tile + (k1 * Y2 + n2) * 8 + (rp ^ (((k1 ^ n2) & 1) << 2)), o);
                    }
                }
            }
            __syncwarp();
            // last inverse y pass + bracket + first forward y pass: lanes = (k1 = 8*rr + lane/4, rql = lane%4)
#pragma unroll 1
            for (int rr = 0; rr < (Y1 + 7) / 8; ++rr) {
                const int k1 = 8 * rr + (lane >> 2), rql = lane & 3;
                if (k1 < Y1) {
                    c2 c[Y2];
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        const int ra = h * (NX / 4) + 4 * qg + rql;
                        c2 v[Y2];
#pragma unroll
                        for (int n2 = 0; n2 < Y2; ++n2)
                            v[n2] = ld_quad(tile + (k1 * Y2 + n2) * 8 + ((h * 4 + rql) ^ (((k1 ^ n2) & 1) << 2)));
                        dft2<Y2, +1>(v);
#pragma unroll
                        for (int k2 = 0; k2 < Y2; ++k2) {
                            const float4 d = __ldg(dchi + (size_t)(k1 * Y2 + k2) * (NX / 2) + ra);
                            const u64 b = fma2(pk2(d.z, d.w), v[k2].re, mul2(pk2(d.x, d.y), v[k2].im));
                            if (h == 0) c[k2].re = b; else c[k2].im = b;
                        }
                    }
                    dft2<Y2, -1>(c);
#pragma unroll
                    for (int d = 0; d < Y2; ++d) {
                        c2 o = c[d];
                        if (d != 0) { const float2 w = twy[k1 * d]; o = cmul_s(o, w.x, -w.y); }
                        st_quad(tile + (k1 * Y2 + d) * 8 + (rql ^ (((k1 ^ d) & 1) << 2)), o);
                    }
                }
            }
            __syncwarp();
            // last forward y pass + 2/3 truncation + separation of the packed rows: lanes = (dd, rql)
#pragma unroll 1
            for (int rr = 0; rr < ((Y2 / 2 + 1) + 7) / 8; ++rr) {
                const int dd = 8 * rr + (lane >> 2), rql = lane & 3;
                if (dd < Y2 / 2 + 1) {
                    const int d0 = dd, d1 = (Y2 - dd) % Y2;
                    c2 u0[Y1], u1[Y1];
#pragma unroll
                    for (int a = 0; a < Y1; ++a) u0[a] = ld_quad(tile + (a * Y2 + d0) * 8 + (rql ^ (((a ^ d0) & 1) << 2)));
                    dft2<Y1, -1>(u0);
                    if (d1 != d0) {
#pragma unroll
                        for (int a = 0; a < Y1; ++a) u1[a] = ld_quad(tile + (a * Y2 + d1) * 8 + (rql ^ (((a ^ d1) & 1) << 2)));
                        dft2<Y1, -1>(u1);
                    } else {
#pragma unroll
                        for (int a = 0; a < Y1; ++a) u1[a] = u0[a];
                    }
                    float* __restrict__ W0 = W + (4 * qg + rql) * RS;
                    const u64 half = bc2(0.5f);
                    auto emit = [&](int k, c2 A, c2 B) {
                        const u64 r0 = mul2(add2(A.re, B.re), half), i0 = mul2(sub2(A.im, B.im), half);
                        const u64 r1 = mul2(add2(A.im, B.im), half), i1 = mul2(sub2(B.re, A.re), half);
                        float* d = W0 + ((k & 1) ? NP : 0) + (k >> 1);
                        float xa, xb;
                        upk2(r0, xa, xb); d[0] = xa; d[(NX / 2) * RS] = xb;
                        upk2(i0, xa, xb); d[IM] = xa; d[IM + (NX / 2) * RS] = xb;
                        upk2(r1, xa, xb); d[(NX / 4) * RS] = xa; d[(3 * NX / 4) * RS] = xb;
                        upk2(i1, xa, xb); d[IM + (NX / 4) * RS] = xa; d[IM + (3 * NX / 4) * RS] = xb;
                    };
#pragma unroll
                    for (int cc = 0; cc <= Q / Y2; ++cc) {
                        {
                            const int k = d0 + Y2 * cc;
                            if (k <= Q) emit(k, u0[cc], (d0 == 0) ? u1[(Y1 - cc) % Y1] : u1[Y1 - 1 - cc]);
                        }
                        if (d1 != d0) {
                            const int k = d1 + Y2 * cc;
                            if (k <= Q) emit(k, u1[cc], u0[Y1 - 1 - cc]);
                        }
                    }
                }
            }
            __syncwarp();
        }
        __syncthreads();                       // B: all rows done; tiles idle, W holds the forward x input

        // prefetch the raw planes of this CTA's next unit into the idle tile region
        if (threadIdx.x == 0 && unit + (int)gridDim.x < nunits) issue_load(unit + gridDim.x);

        // ---------------- a6 (x part) + a7, warp-local per kept ky pair
        float2* __restrict__ out = p.bhat + (size_t)unit * NK;
        for (int tp = warp; tp < NP; tp += C::NW) {
            if (lane < X1) {
                const int a = lane;
                float* __restrict__ Wa = W + a * X2 * RS + tp;
                c2 v[X2];
#pragma unroll
                for (int b = 0; b < X2; ++b) {
                    const float* sp = Wa + b * RS;
                    v[b].re = pk2(sp[0], sp[NP]); v[b].im = pk2(sp[IM], sp[IM + NP]);
                }
                dft2<X2, -1>(v);
#pragma unroll
                for (int d = 0; d < X2; ++d) {
                    c2 o = v[d];
                    if (d != 0) { const float2 w = twx[a * d]; o = cmul_s(o, w.x, -w.y); }
                    float ra, rb, ia, ib;
                    upk2(o.re, ra, rb); upk2(o.im, ia, ib);
                    float* dst = Wa + d * RS;
                    dst[0] = ra; dst[NP] = rb; dst[IM] = ia; dst[IM + NP] = ib;
                }
            }
            __syncwarp();
            if (lane < X2) {
                const int d = lane;
                const float* __restrict__ Wa = W + d * RS + tp;
                c2 v[X1];
#pragma unroll
                for (int a = 0; a < X1; ++a) {
                    const float* sp = Wa + a * X2 * RS;
                    v[a].re = pk2(sp[0], sp[NP]); v[a].im = pk2(sp[IM], sp[IM + NP]);
                }
                dft2<X1, -1>(v);
                const u64 sc = bc2(p.scale);
#pragma unroll
                for (int cc = 0; cc < X1; ++cc) {
                    if (cc * X2 <= K || cc * X2 + X2 - 1 >= NX - K) {
                        const int n = d + X2 * cc;
                        int i = -1;
                        if (n <= K) i = n;
                        else if (n >= NX - K) i = n - NX + NAKX;
                        if (i >= 0) {
                            float ra, rb, ia, ib;
                            upk2(mul2(v[cc].re, sc), ra, rb); upk2(mul2(v[cc].im, sc), ia, ib);
                            *reinterpret_cast<float4*>(out + i * NAKY + 2 * tp) = make_float4(ra, ia, rb, ib);
                        }
                    }
                }
            }
            __syncwarp();
        }
        // ---- publish this node's Bhat plane; the barrier also frees W for the next unit
        __syncthreads();                       // D
        if (threadIdx.x == 0) { __threadfence(); atomicAdd(p.count + (s * p.Nm + m) * p.Nz + z, 1u); }
    }
}

}  // namespace gx
