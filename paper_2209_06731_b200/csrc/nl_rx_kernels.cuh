// nl_rx_kernels.cuh -- "rx" kernel family of the nonlinear E×B term (sm_100a, fp32): packed-FP32 x passes,
// one-thread-per-row y direction, inverse Laguerre transform fused into the same kernel.
// PAPER.md lines 646-655 (App. D Eq. D1 line 1); rows a1-a8 of SURVEY.md section 8(a).
//
// What changed against the "row" family (nl_row_kernels.cuh; r01c capture: issue-bound while it runs, the x
// passes hold half of its instructions, a separate inverse-Laguerre kernel behind a 21 MB workspace):
//
//  * The two real fields d_x f and d_y f are no longer one complex field on 2*naky-1 columns.  Their
//    half-spectra P = i kx f and R = i ky f (ky >= 0 only: naky columns) ride in the two lanes of packed
//    FP32 registers (dft_packed.cuh): one x transform of packed values replaces the two transforms of the
//    columns +ky and -ky, with shared loads, addresses and twiddles, and every butterfly, rotation and
//    twiddle product is an FADD2 / FMUL2 / FFMA2.  The plane buffer W4[x][ky] holds float4
//    (P.re, R.re, P.im, R.im): same bytes as before, 128-bit accesses.
//  * y direction of a row, one thread: the two real 64-point inverse transforms are ONE packed 32-point
//    complex transform (even/odd sample packing, again both fields in the two lanes), then the bracket, then
//    the real forward transform (32-point complex + split) as in the row family.
//  * Forward x passes: two neighbouring ky columns per packed value (naky/2 column pairs).
//  * a8: the CTA that completes the last of the J nodes of an (s,m,z) (arrival counter) forms
//    out_l = - sum_j Tinv[l][j] Bhat_j for that (s,m,z) itself from the node planes, which are still in L2;
//    there is no third kernel and no spin-waiting grid.
//  * The chi planes are stored as float4 (d_x chi, d_y chi) at y = 2i and 2i+1: one 128-bit load per two
//    y points in the bracket.
//
// Every phase is a __host__ __device__ function of the thread index: tests/host_emul/rx_emul.cu runs the
// same code on the CPU, thread by thread, over bounds- and hazard-checked arrays (profiles/r02_sanitizer.md).
#pragma once
#include "dft_packed.cuh"
#include "nl_kernels.cuh"

namespace gx {

// shared / global accessors: raw pointers on the device, checked pointers in tests/host_emul
template <class T> GX_HD T ld(const T* p, int i) { return p[i]; }
template <class T> GX_HD T ld(T* p, int i) { return p[i]; }
template <class T> GX_HD void st(T* p, int i, const T& v) { p[i] = v; }

template <int NX_, int NY_, int RX1_, int RX2_, int NT_, int MINB_>
struct RxCfg {
    static constexpr int NX = NX_, NY = NY_, RX1 = RX1_, RX2 = RX2_, NT = NT_, MINB = MINB_;
    static constexpr int K = (NX - 1) / 3, Q = (NY - 1) / 3;
    static constexpr int NAKX = 2 * K + 1, NAKY = Q + 1, NK = NAKX * NAKY, NK2 = NK / 2;
    static constexpr int NP = NAKY / 2;              // ky column pairs of the forward x passes
    // W4 row stride in float4 = NAKY (even) with the slots of a row XOR-swizzled by bit 2 of the row: rows r..r+7
    // then hit eight different 16-byte bank groups for a fixed ky (row phase), and a row stays a permutation of
    // consecutive slots (x passes) -- conflict-free without the padding column (3 KB per plane buffer)
    static constexpr int RS = NAKY;
    GX_HD static int widx(int row, int q) { return row * RS + (q ^ ((row >> 2) & 1)); }
    static constexpr int H = NY / 2;                 // complex length behind the real y transforms
    static constexpr int W4_ELEMS = NX * RS;         // float4
    static constexpr int S_ELEMS = NK;               // float2; S sits at the start of the dynamic shared memory
    static constexpr int STAGE_BYTES = S_ELEMS * 8 + W4_ELEMS * 16;
    static constexpr int CAP = STAGE_BYTES / (NK * 8);            // raw Laguerre planes per staging chunk
    static constexpr int SMEM_BYTES = STAGE_BYTES + NX * 8;
    static constexpr int PER = (NK2 + NT - 1) / NT;              // float4 slots of a compact plane per thread
    static constexpr unsigned zero_mask(int R1, int R2, int N, int KK) {
        unsigned m = 0;
        for (int n1 = 0; n1 < R1; ++n1)
            if (!(n1 * R2 <= KK || n1 * R2 + R2 - 1 >= N - KK)) m |= 1u << n1;
        return m;
    }
    static constexpr unsigned ZMX = zero_mask(RX1, RX2, NX, K);
    static_assert(NY == 64, "the single-thread y transforms are written for 64 points");
    static_assert(RX1 * RX2 == NX && NAKY % 2 == 0, "radix split / ky column pairs");
    static_assert(CAP >= 2, "staging needs room for two raw planes");
    static_assert(SMEM_BYTES <= 232448, "plane does not fit in shared memory");
    static_assert(H - Q <= Q + 1 && Q < H, "every bin of the half-length transform has an input, no Nyquist mode");
};

GX_HD pk::c2 c2_from(float4 f) { return pk::make_c2(pk::pk2(f.x, f.y), pk::pk2(f.z, f.w)); }
GX_HD float4 f4_from(pk::c2 v) {
    float4 f;
    pk::upk2(v.re, f.x, f.y);
    pk::upk2(v.im, f.z, f.w);
    return f;
}

// ------------------------------------------------------------------------------------------------
// a2: S[slot] (+)= sum_l coef[l] raw_l[slot] over the planes of one staging chunk, in place: plane 0 of the
// first chunk lands on S itself, so a thread only ever overwrites slots it has just read.
template <class C, int NT = C::NT, class P4>
GX_HD void rx_combine(int tid, P4 stage4, const float* coef, int l0, int nl, bool first) {
    // stage4: float4 view of the staging region; plane at slot index sl occupies [sl*NK2, (sl+1)*NK2)
    constexpr int PER = (C::NK2 + NT - 1) / NT;
#pragma unroll
    for (int u = 0; u < PER; ++u) {
        const int slot = u * NT + tid;
        if (slot < C::NK2) {
            float4 acc = first ? make_float4(0.f, 0.f, 0.f, 0.f) : ld(stage4, slot);
            for (int l = 0; l < nl; ++l) {
                const float t = coef[l0 + l];
                const float4 f = ld(stage4, (first ? l : l + 1) * C::NK2 + slot);
                acc.x = fmaf(t, f.x, acc.x);
                acc.y = fmaf(t, f.y, acc.y);
                acc.z = fmaf(t, f.z, acc.z);
                acc.w = fmaf(t, f.w, acc.w);
            }
            st(stage4, slot, acc);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// a3 + a4 (x part).  Item (n2, q): inputs f(n, q), n = n1*R2 + n2, of the compact plane S (kept rows only:
// class of n1 resolved at compile time, at most two n1 decided by n2), lanes P = i kx f and R = i ky f,
// DFT_R1 over n1, twiddle, W4[(k1*R2 + n2)][q].
template <class C, class P2>
GX_HD void rx_xi1_load(P2 S, int n2, int q, float dkx, float ky, pk::c2 (&v)[C::RX1]) {
    constexpr int NX = C::NX, K = C::K, NAKY = C::NAKY, NAKX = C::NAKX, R1 = C::RX1, R2 = C::RX2;
#pragma unroll
    for (int n1 = 0; n1 < R1; ++n1) {
        const int lo = n1 * R2, hi = n1 * R2 + R2 - 1;           // range of n over n2 (compile time)
        const bool allP = hi <= K, someP = lo <= K;              // kept with kx >= 0
        const bool allN = lo >= NX - K, someN = hi >= NX - K;    // kept with kx < 0
        v[n1] = pk::czero();
        if (someP || someN) {
            float2 f = make_float2(0.f, 0.f);
            float kx = 0.f;
            if (someP && (allP || lo + n2 <= K)) {
                f = ld(S, (lo + n2) * NAKY + q);
                kx = dkx * (float)(lo + n2);
            }
            if (someN && (allN || lo + n2 >= NX - K)) {
                f = ld(S, (lo + n2 - NX + NAKX) * NAKY + q);
                kx = dkx * (float)(lo + n2 - NX);
            }
            // P = i kx f = (-kx f.im, kx f.re),  R = i ky f = (-ky f.im, ky f.re)
            v[n1] = pk::make_c2(pk::mul2(pk::bc2(f.y), pk::pk2(-kx, -ky)), pk::mul2(pk::bc2(f.x), pk::pk2(kx, ky)));
        }
    }
}
template <class C, class P4, class PT>
GX_HD void rx_xi1_store(P4 W4, PT twx, int n2, int q, const pk::c2 (&v)[C::RX1]) {
#pragma unroll
    for (int k1 = 0; k1 < C::RX1; ++k1) {
        pk::c2 o = v[k1];
        if (k1 > 0) {
            const float2 w = ld(twx, n2 * k1);
            o = pk::cmul_s(o, w.x, w.y);
        }
        st(W4, C::widx(k1 * C::RX2 + n2, q), f4_from(o));
    }
}
// single-item form (fewer registers; the x workers of the pipelined kernel run it with their own thread count)
template <class C, int NT, class P2, class P4, class PT>
GX_HD void rx_x_inverse_pass1_single(int tid, P2 S, P4 W4, PT twx, float dkx, float dky) {
    constexpr int NAKY = C::NAKY, R1 = C::RX1, R2 = C::RX2, NITEM = R2 * NAKY;
    for (int t = tid; t < NITEM; t += NT) {
        const int n2 = t / NAKY, q = t - n2 * NAKY;
        pk::c2 v[R1];
        rx_xi1_load<C>(S, n2, q, dkx, dky * (float)q, v);
        pk::dft<R1, +1, C::ZMX>(v);
        rx_xi1_store<C>(W4, twx, n2, q, v);
    }
}
template <class C, int NT, class P4>
GX_HD void rx_x_inverse_pass2_single(int tid, P4 W4) {
    constexpr int NAKY = C::NAKY, R1 = C::RX1, R2 = C::RX2, NITEM = R1 * NAKY;
    for (int t = tid; t < NITEM; t += NT) {
        const int k1 = t / NAKY, q = t - k1 * NAKY;
        pk::c2 v[R2];
#pragma unroll
        for (int n2 = 0; n2 < R2; ++n2) v[n2] = c2_from(ld(W4, C::widx(k1 * R2 + n2, q)));
        pk::dft<R2, +1>(v);
#pragma unroll
        for (int k2 = 0; k2 < R2; ++k2) st(W4, C::widx(k1 * R2 + k2, q), f4_from(v[k2]));
    }
}

template <class C, class P2, class P4, class PT>
GX_HD void rx_x_inverse_pass1(int tid, P2 S, P4 W4, PT twx, float dkx, float dky) {
    constexpr int NAKY = C::NAKY, R1 = C::RX1, R2 = C::RX2, NT = C::NT, NITEM = R2 * NAKY;
    for (int t0 = tid; t0 < NITEM; t0 += 2 * NT) {
        // items t0 and t0 + NT together: two independent dependency chains per thread (the pass is latency-bound:
        // r02 phase benchmark); a missing second item repeats the first and is not stored
        const int t1 = t0 + NT;
        const bool has1 = t1 < NITEM;
        const int ta = t0, tb = has1 ? t1 : t0;
        const int n2a = ta / NAKY, qa = ta - n2a * NAKY, n2b = tb / NAKY, qb = tb - n2b * NAKY;
        if ((t1 & ~31) < NITEM) {                  // some lane of this warp has a second item (warp-uniform)
            pk::c2 va[R1], vb[R1];
            rx_xi1_load<C>(S, n2a, qa, dkx, dky * (float)qa, va);
            rx_xi1_load<C>(S, n2b, qb, dkx, dky * (float)qb, vb);
            pk::dft<R1, +1, C::ZMX>(va);
            pk::dft<R1, +1, C::ZMX>(vb);
            rx_xi1_store<C>(W4, twx, n2a, qa, va);
            if (has1) rx_xi1_store<C>(W4, twx, n2b, qb, vb);
        } else {
            pk::c2 va[R1];
            rx_xi1_load<C>(S, n2a, qa, dkx, dky * (float)qa, va);
            pk::dft<R1, +1, C::ZMX>(va);
            rx_xi1_store<C>(W4, twx, n2a, qa, va);
        }
    }
}

// Item (k1, q): DFT_R2 over n2; position k1*R2 + k2 <- x = k1 + R1*k2.  Two items per thread as above.
template <class C, class P4>
GX_HD void rx_x_inverse_pass2(int tid, P4 W4) {
    constexpr int NAKY = C::NAKY, R1 = C::RX1, R2 = C::RX2, NT = C::NT, NITEM = R1 * NAKY;
    for (int t0 = tid; t0 < NITEM; t0 += 2 * NT) {
        const int t1 = t0 + NT;
        const bool has1 = t1 < NITEM;
        const int ta = t0, tb = has1 ? t1 : t0;
        const int k1a = ta / NAKY, qa = ta - k1a * NAKY, k1b = tb / NAKY, qb = tb - k1b * NAKY;
        if ((t1 & ~31) < NITEM) {                  // some lane of this warp has a second item (warp-uniform)
            pk::c2 va[R2], vb[R2];
#pragma unroll
            for (int n2 = 0; n2 < R2; ++n2) {
                va[n2] = c2_from(ld(W4, C::widx(k1a * R2 + n2, qa)));
                vb[n2] = c2_from(ld(W4, C::widx(k1b * R2 + n2, qb)));
            }
            pk::dft<R2, +1>(va);
            pk::dft<R2, +1>(vb);
#pragma unroll
            for (int k2 = 0; k2 < R2; ++k2) st(W4, C::widx(k1a * R2 + k2, qa), f4_from(va[k2]));
            if (has1) {
#pragma unroll
                for (int k2 = 0; k2 < R2; ++k2) st(W4, C::widx(k1b * R2 + k2, qb), f4_from(vb[k2]));
            }
        } else {
            pk::c2 va[R2];
#pragma unroll
            for (int n2 = 0; n2 < R2; ++n2) va[n2] = c2_from(ld(W4, C::widx(k1a * R2 + n2, qa)));
            pk::dft<R2, +1>(va);
#pragma unroll
            for (int k2 = 0; k2 < R2; ++k2) st(W4, C::widx(k1a * R2 + k2, qa), f4_from(va[k2]));
        }
    }
}

// ------------------------------------------------------------------------------------------------
// a6 (x part): forward x transform of the column pairs (lane 0 = ky 2p, lane 1 = ky 2p+1).
// Item (a, p): DFT_R2 over b of W4[(a*R2 + b)][p], twiddle e^{-2 pi i a d / NX}, back in place.
template <class C, int NT = C::NT, class P4, class PT>
GX_HD void rx_x_forward_pass1(int tid, P4 W4, PT twx) {
    constexpr int NP = C::NP, R1 = C::RX1, R2 = C::RX2;
    for (int t = tid; t < R1 * NP; t += NT) {
        const int a = t / NP, pp = t - a * NP;
        pk::c2 v[R2];
#pragma unroll
        for (int b = 0; b < R2; ++b) v[b] = c2_from(ld(W4, C::widx(a * R2 + b, pp)));
        pk::dft<R2, -1>(v);
#pragma unroll
        for (int d = 0; d < R2; ++d) {
            pk::c2 o = v[d];
            if (d > 0) {
                const float2 w = ld(twx, a * d);
                o = pk::cmul_s(o, w.x, -w.y);
            }
            st(W4, C::widx(a * R2 + d, pp), f4_from(o));
        }
    }
}

// Item (d, p): DFT_R1 over a; kept rows n = d + R2*cc (|kx| <= K: a7) times `scale` to the compact plane
// out4 (float4 = two neighbouring ky of one kx row; NAKY even).
template <class C, int NT = C::NT, class P4, class PO>
GX_HD void rx_x_forward_pass2(int tid, P4 W4, PO out4, float scale) {
    constexpr int NX = C::NX, K = C::K, NAKX = C::NAKX, NP = C::NP, R1 = C::RX1, R2 = C::RX2;
    for (int t = tid; t < R2 * NP; t += NT) {
        const int d = t / NP, pp = t - d * NP;
        pk::c2 v[R1];
#pragma unroll
        for (int a = 0; a < R1; ++a) v[a] = c2_from(ld(W4, C::widx(a * R2 + d, pp)));
        pk::dft<R1, -1>(v);
#pragma unroll
        for (int cc = 0; cc < R1; ++cc) {
            if (cc * R2 <= K || cc * R2 + R2 - 1 >= NX - K) {
                const int n = d + R2 * cc;
                int i = -1;
                if (n <= K) i = n;
                else if (n >= NX - K) i = n - NX + NAKX;
                if (i >= 0) {
                    const float4 f = f4_from(v[cc]);     // (re0, re1, im0, im1)
                    st(out4, i * NP + pp, make_float4(f.x * scale, f.z * scale, f.y * scale, f.w * scale));
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// y direction of one x row, one thread.
//
// Real inverse transforms of the two fields at once (lanes P, R).  With the kept coefficients C_q, q = 0..Q,
// C_{-q} = conj C_q, x[n] = sum_q C_q e^{2 pi i q n / NY} is real; its even and odd samples are the real and
// imaginary parts of the H = NY/2 point complex inverse transform of
//      Z_k = E_k + i O_k,   E_k = C_k + conj C_{H-k},   O_k = w^k (C_k - conj C_{H-k}),   w = e^{2 pi i / NY},
// where C_k = 0 for k > Q (2/3 rule): bins with one contributor cost one packed complex multiplication by the
// constant 1 + i w^k (or its mirror), bins with two cost ten packed operations.  Im C_0 (rounding noise of a
// Hermitian ky = 0 column) is dropped.
template <class C>
GX_HD void rx_c2r_prep(const pk::c2 (&Cq)[C::NAKY], pk::c2 (&Z)[C::H]) {
    constexpr int H = C::H, Q = C::Q, NY = C::NY;
#pragma unroll
    for (int k = 0; k < H; ++k) {
        const int h = H - k;
        const bool has_lo = k <= Q, has_hi = k > 0 && h <= Q;
        const double cd = cos192(k * (192 / NY)), sd = sin192(k * (192 / NY));
        if (k == 0) {
            Z[0] = pk::make_c2(Cq[0].re, Cq[0].re);
        } else if (has_lo && !has_hi) {
            Z[k] = pk::cmul_s(Cq[k], (float)(1.0 - sd), (float)cd);                 // C_k (1 + i w^k)
        } else if (!has_lo && has_hi) {
            Z[k] = pk::cmul_conj_s(Cq[h < C::NAKY ? h : 0], (float)(1.0 + sd), (float)(-cd));   // conj(C_{H-k}) (1 - i w^k)
        } else {
            const pk::c2 a = Cq[k <= Q ? k : 0], b = Cq[h < C::NAKY ? h : 0];
            const pk::c2 E = pk::make_c2(pk::add2(a.re, b.re), pk::sub2(a.im, b.im));
            const pk::c2 D = pk::make_c2(pk::sub2(a.re, b.re), pk::add2(a.im, b.im));
            const pk::c2 O = pk::cmul_s(D, (float)cd, (float)sd);
            Z[k] = pk::make_c2(pk::sub2(E.re, O.im), pk::add2(E.im, O.re));
        }
    }
}

GX_HD void prefetch_l1(const void* p) {
#ifdef __CUDA_ARCH__
    asm volatile("prefetch.global.L1 [%0];" ::"l"(p));
#else
    (void)p;
#endif
}
template <class T> GX_HD const void* addr_of(const T* p, int i) { return p + i; }

template <class C, class P4>
GX_HD void rx_row_load(P4 W4, int row, pk::c2 (&Cq)[C::NAKY]) {
#pragma unroll
    for (int q = 0; q < C::NAKY; ++q) Cq[q] = c2_from(ld(W4, C::widx(row, q)));
}

// a4 (y part) + a5 + a6 (y part) + a7 (ky <= Q) for the rows of this thread.  dchi4[i*NX + row] holds
// (d_x chi, d_y chi) at y = 2i and y = 2i+1 of the row.
template <class C, class P4, class PD>
GX_HD void rx_row_bracket(int tid, P4 W4, PD dchi4) {
    constexpr int NX = C::NX, NY = C::NY, H = C::H, Q = C::Q, NP = C::NP;
    constexpr int A = 8, B = 4;                    // H = A*B: second stage in groups of B outputs i = k1 + A*k2
    static_assert(A * B == H, "split of the half-length transform");
    for (int row = tid; row < NX; row += C::NT) {
        // chi pairs of output group k1+1 are requested while group k1 is transformed, groups k1+2, k1+3 are
        // prefetched towards L1: the L2 latency of dchi hides behind the butterflies
        float4 d[B], dn[B];
#pragma unroll
        for (int k2 = 0; k2 < B; ++k2) d[k2] = ld(dchi4, (A * k2) * NX + row);
#pragma unroll
        for (int k2 = 0; k2 < B; ++k2) {
            prefetch_l1(addr_of(dchi4, (1 + A * k2) * NX + row));
            prefetch_l1(addr_of(dchi4, (2 + A * k2) * NX + row));
        }
        pk::c2 Y[H];
        {
            pk::c2 Cq[C::NAKY], Z[H];
            rx_row_load<C>(W4, row, Cq);
            rx_c2r_prep<C>(Cq, Z);
            pk::dft_split_col<H, A, B, +1, 0ull, 0>(Z, Y);
        }
        float b[NY];
#pragma unroll
        for (int k1 = 0; k1 < A; ++k1) {
            if (k1 + 1 < A) {
#pragma unroll
                for (int k2 = 0; k2 < B; ++k2) dn[k2] = ld(dchi4, (k1 + 1 + A * k2) * NX + row);
            }
            if (k1 + 3 < A) {
#pragma unroll
                for (int k2 = 0; k2 < B; ++k2) prefetch_l1(addr_of(dchi4, (k1 + 3 + A * k2) * NX + row));
            }
            pk::c2 u[B];
#pragma unroll
            for (int n2 = 0; n2 < B; ++n2) u[n2] = Y[k1 * B + n2];
            pk::Dft<B, +1, 0ull>::run(u);
#pragma unroll
            for (int k2 = 0; k2 < B; ++k2) {
                const int i = k1 + A * k2;             // samples y = 2i (real parts) and 2i+1 (imaginary parts)
                float p0, r0, p1, r1;
                pk::upk2(u[k2].re, p0, r0);
                pk::upk2(u[k2].im, p1, r1);
                b[2 * i] = fmaf(d[k2].y, p0, -d[k2].x * r0);          // d_y chi d_x g - d_x chi d_y g
                b[2 * i + 1] = fmaf(d[k2].w, p1, -d[k2].z * r1);
                d[k2] = dn[k2];
            }
        }
        // real forward transform: H-point complex transform of the even/odd packing + split, kept ky only
        float2 zc[H];
#pragma unroll
        for (int i = 0; i < H; ++i) zc[i] = make_float2(b[2 * i], b[2 * i + 1]);
        dft<H, -1>(zc);
        float2 F[C::NAKY];
#pragma unroll
        for (int k = 0; k <= Q; ++k) {
            const float2 a = zc[k], c = zc[(H - k) % H];
            const float2 e = make_float2(0.5f * (a.x + c.x), 0.5f * (a.y - c.y));
            const float2 o = make_float2(0.5f * (a.y + c.y), 0.5f * (c.x - a.x));
            F[k] = cadd(e, twiddle<NY, -1>(o, k));
        }
#pragma unroll
        for (int pp = 0; pp < NP; ++pp)
            st(W4, C::widx(row, pp), make_float4(F[2 * pp].x, F[2 * pp + 1].x, F[2 * pp].y, F[2 * pp + 1].y));
    }
}

// chi planes: y inverse only, result stored as float4 (d_x chi, d_y chi) at y = 2i, 2i+1.
template <class C, class P4, class PD>
GX_HD void rx_row_chi(int tid, P4 W4, PD dchi4) {
    constexpr int NX = C::NX, H = C::H;
    for (int row = tid; row < NX; row += C::NT) {
        pk::c2 Z[H];
        {
            pk::c2 Cq[C::NAKY];
            rx_row_load<C>(W4, row, Cq);
            rx_c2r_prep<C>(Cq, Z);
        }
        pk::dft<H, +1>(Z);
#pragma unroll
        for (int i = 0; i < H; ++i) st(dchi4, i * NX + row, f4_from(Z[i]));
    }
}

// node planes written by other SMs during this kernel: read through L2 (ld.global.cg), never through L1
struct CgPtr { const float4* p; };
GX_HD float4 ld(CgPtr c, int i) {
#ifdef __CUDA_ARCH__
    return __ldcg(c.p + i);
#else
    return c.p[i];
#endif
}

// a8 for one (s,m,z): out_l = sum_j Ti[l][j] Bhat_j with Ti = -Tinv (out = -N), float4 = two coefficients.
// bh4: node plane j at bh4 + j*jstride4; out4: moment plane l at out4 + l*lstride4.
template <class C, class PB, class PO>
GX_HD void rx_laguerre_inverse(int tid, PB bh4, int jstride4, PO out4, int lstride4, const float* Ti, int Nl, int J) {
    // two slots of the plane and up to JU node planes per round trip: 2*JU independent 16-byte loads in flight
    constexpr int JU = 8, NT = C::NT, NK2 = C::NK2;
    for (int slot0 = tid; slot0 < NK2; slot0 += 2 * NT) {
        const int slot1 = slot0 + NT;
        const bool has1 = slot1 < NK2;
        for (int l0 = 0; l0 < Nl; l0 += 4) {
            float4 acc[2][4];
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
                for (int dl = 0; dl < 4; ++dl) acc[h][dl] = make_float4(0.f, 0.f, 0.f, 0.f);
            for (int j0 = 0; j0 < J; j0 += JU) {
                float4 bv[2][JU];
#pragma unroll
                for (int jj = 0; jj < JU; ++jj) {
                    const bool on = j0 + jj < J;
                    bv[0][jj] = on ? ld(bh4, (j0 + jj) * jstride4 + slot0) : make_float4(0.f, 0.f, 0.f, 0.f);
                    bv[1][jj] = (on && has1) ? ld(bh4, (j0 + jj) * jstride4 + slot1) : make_float4(0.f, 0.f, 0.f, 0.f);
                }
#pragma unroll
                for (int jj = 0; jj < JU; ++jj) {
                    if (j0 + jj < J) {
#pragma unroll
                        for (int dl = 0; dl < 4; ++dl) {
                            const float t = (l0 + dl < Nl) ? Ti[(l0 + dl) * J + j0 + jj] : 0.f;
#pragma unroll
                            for (int h = 0; h < 2; ++h) {
                                acc[h][dl].x = fmaf(t, bv[h][jj].x, acc[h][dl].x);
                                acc[h][dl].y = fmaf(t, bv[h][jj].y, acc[h][dl].y);
                                acc[h][dl].z = fmaf(t, bv[h][jj].z, acc[h][dl].z);
                                acc[h][dl].w = fmaf(t, bv[h][jj].w, acc[h][dl].w);
                            }
                        }
                    }
                }
            }
#pragma unroll
            for (int dl = 0; dl < 4; ++dl)
                if (l0 + dl < Nl) {
                    st(out4, (l0 + dl) * lstride4 + slot0, acc[0][dl]);
                    if (has1) st(out4, (l0 + dl) * lstride4 + slot1, acc[1][dl]);
                }
        }
    }
}

#ifdef __CUDACC__
// ================================================================================================
// a1 + a3 + a4 for the potential: (d_x chi, d_y chi) of chi_{s,z,j} = M_{s,z,j} Phi_z on the real grid.
template <class C>
__global__ void __launch_bounds__(C::NT, C::MINB) chi_planes_rx_kernel(const NlParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2* S = reinterpret_cast<float2*>(smem_raw);
    float4* W4 = reinterpret_cast<float4*>(smem_raw + C::S_ELEMS * 8);
    float2* twx = reinterpret_cast<float2*>(smem_raw + C::STAGE_BYTES);
    const int tid = threadIdx.x;
    const int unit = blockIdx.x;                 // (s*Nz + z)*J + j
    const int z = (unit / p.J) % p.Nz;
    const float2* __restrict__ phi = p.phi + (size_t)(p.phi_by_unit ? unit : z) * C::NK;
    const float* __restrict__ M = p.M + (size_t)(p.M_shared ? 0 : unit) * C::NK;
    pdl_launch_dependents();        // the bracket kernel's prologue (a2-a4 x part) does not read dchi
    for (int i = tid; i < C::NX; i += C::NT) twx[i] = p.twx[i];
    for (int i = tid; i < C::NK; i += C::NT) {
        const float2 f = __ldg(phi + i);
        const float m = __ldg(M + i);
        S[i] = make_float2(f.x * m, f.y * m);
    }
    __syncthreads();
    rx_x_inverse_pass1<C>(tid, (const float2*)S, W4, (const float2*)twx, p.dkx, p.dky);
    __syncthreads();
    rx_x_inverse_pass2<C>(tid, W4);
    __syncthreads();
    rx_row_chi<C>(tid, (const float4*)W4, reinterpret_cast<float4*>(p.dchi) + (size_t)unit * C::H * C::NX);
}

// ================================================================================================
// a2-a8 for one (s,m,z,j): Bhat_j(k) = F_k[ d_y chi d_x gt - d_x chi d_y gt ], 2/3-rule truncated; the last
// node unit of an (s,m,z) to arrive also writes out_l = - sum_j Tinv[l][j] Bhat_j for that (s,m,z).
template <class C>
__global__ void __launch_bounds__(C::NT, C::MINB) bracket_rx_kernel(const NlParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2* S = reinterpret_cast<float2*>(smem_raw);
    float4* stage4 = reinterpret_cast<float4*>(smem_raw);
    float4* W4 = reinterpret_cast<float4*>(smem_raw + C::S_ELEMS * 8);
    float2* twx = reinterpret_cast<float2*>(smem_raw + C::STAGE_BYTES);
    constexpr int NK = C::NK;
    const int tid = threadIdx.x;

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
    __shared__ float Ti[16 * 23];
    __shared__ int last_flag;
    unsigned bar_parity = 0;
    GX_PHASE(0);
    if (tid == 0) mbar_init(&stage_bar, 1);
    if (tid < p.Nl) Tsh[tid] = __ldg(p.T + j * p.Nl + tid);
    for (int i = tid; i < p.Nl * p.J; i += C::NT) Ti[i] = -__ldg(p.Tinv + i);          // out = -N
    for (int i = tid; i < C::NX; i += C::NT) twx[i] = p.twx[i];
    __syncthreads();
    pdl_launch_dependents();
    // ---- a2: forward Laguerre transform l -> node j, fused into the TMA-staged load (cp.async.bulk + mbarrier)
    for (int l0 = 0; l0 < p.Nl;) {
        const bool first = l0 == 0;
        const int nl = min(first ? C::CAP : C::CAP - 1, p.Nl - l0);
        if (tid == 0) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            mbar_expect_tx(&stage_bar, (unsigned)(nl * NK * sizeof(float2)));
            for (int l = 0; l < nl; ++l)
                bulk_g2s(S + (size_t)(first ? l : l + 1) * NK, g0 + (size_t)(l0 + l) * lstride, NK * sizeof(float2), &stage_bar);
        }
        mbar_wait(&stage_bar, bar_parity);
        bar_parity ^= 1u;
        rx_combine<C>(tid, stage4, Tsh, l0, nl, first);
        __syncthreads();                                         // chunk consumed / S complete
        l0 += nl;
    }
    GX_PHASE(1);
    // ---- a3 + a4 (x part)
    rx_x_inverse_pass1<C>(tid, (const float2*)S, W4, (const float2*)twx, p.dkx, p.dky);
    __syncthreads();
    rx_x_inverse_pass2<C>(tid, W4);
    __syncthreads();
    GX_PHASE(2);
    pdl_wait();                     // chi planes of this call are complete and visible from here on
    GX_PHASE(3);
    // ---- a4 (y part) + a5 + a6 (y part) + a7 (ky)
    rx_row_bracket<C>(tid, W4, reinterpret_cast<const float4*>(p.dchi) + (size_t)szj * C::H * C::NX);
    __syncthreads();
    GX_PHASE(4);
    // ---- a6 (x part) + a7 (kx)
    rx_x_forward_pass1<C>(tid, W4, (const float2*)twx);
    __syncthreads();
    rx_x_forward_pass2<C>(tid, (const float4*)W4, reinterpret_cast<float4*>(p.bhat + (size_t)unit * NK), p.scale);
    // ---- a8: publish this node plane (release: stores -> barrier -> fence -> atomic); the unit that completes
    // the (s,m,z) resets the counter and does the sum over j (a handle runs one call at a time)
    __syncthreads();
    GX_PHASE(5);
    if (tid == 0) {
        __threadfence();
        unsigned* cnt = p.count + (s * p.Nm + m) * p.Nz + z;
        const unsigned old = atomicAdd(cnt, 1u);
        last_flag = (old + 1u == (unsigned)p.J);
        if (last_flag) *cnt = 0u;   // nobody touches this counter again before the next call (stream order)
    }
    __syncthreads();
    if (last_flag) {
        __threadfence();            // acquire side: the other nodes' planes are visible (read through L2 below)
        const int jstride4 = p.Nm * C::NK2;
        const float4* bh4 = reinterpret_cast<const float4*>(p.bhat + ((size_t)((s * p.Nz + z) * p.J) * p.Nm + m) * NK);
        float4* out4 = reinterpret_cast<float4*>(p.out + (((size_t)(s * p.Nm + m) * p.Nl) * p.Nz + z) * NK);
        rx_laguerre_inverse<C>(tid, CgPtr{bh4}, jstride4, out4, (int)(lstride / 2), Ti, p.Nl, p.J);
    }
    GX_PHASE(6);
}

// ================================================================================================
// Persistent form of the same path: ONE kernel per gx_nonlinear_rhs call, one CTA per SM, two independent
// groups of NT threads per CTA (each owns a plane buffer and runs the phases above with named barriers).
//
// Why (r02 captures of bracket_rx_kernel, profiles/r02_rx_ncu.md): (i) with two 6-warp CTAs per SM the warp
// schedulers 0 and 1 carry twice the warps of 2 and 3 (warp w of a CTA lives on scheduler w mod 4; measured
// 1.74x spread of instructions per scheduler) -- twelve warps of one CTA spread 3/3/3/3; (ii) the release
// fence + arrival atomic of a unit (2 k cycles) and the TMA latency of the next unit's planes now overlap:
// the planes of unit u+1 are requested as soon as the plane buffer of unit u is dead, the fence and atomic
// run in thread 0 meanwhile, and the "was I the last node" answer is consumed one unit later; (iii) the chi
// planes are items of the same work list (they come first and never wait), a bracket unit waits for its
// plane's ready flag just before its row phase: no second kernel, no programmatic-dependent-launch chain.
//
// Work list: items [0, n_chi) are chi planes (s,z,j); items [n_chi, n_chi + n_units) bracket units
// ((s,z,j),m).  Group gid takes items gid, gid + G, gid + 2G, ... (G = number of groups in the grid).
// All CTAs are co-resident (grid <= number of SMs) and chi items never wait, so the flag waits cannot deadlock.
__device__ __forceinline__ void group_bar(int grp, int nthreads) {
    asm volatile("bar.sync %0, %1;" ::"r"(grp + 1), "r"(nthreads) : "memory");
}
__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_u32(unsigned* p, unsigned v) {
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

#ifdef GX_PHASE_TIMING
// development builds: per group and per processed item, clock64() at phase boundaries and %globaltimer at the start
static __device__ long long gx_phase2_clk[512 * 8 * 12];
__device__ __forceinline__ long long gx_globaltimer() { long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t; }
#define GX_PHASE2(i) do { if (tid == 0 && gid < 512 && round < 8) gx_phase2_clk[(gid * 8 + round) * 12 + (i)] = ((i) == 0 ? gx_globaltimer() : clock64()); } while (0)
#else
#define GX_PHASE2(i) do { } while (0)
#endif

struct RxUnit { int s, m, z, j, szj; };
__device__ __forceinline__ RxUnit rx_decode(int unit, const NlParams& p) {
    RxUnit u;
    u.m = unit % p.Nm;
    u.szj = unit / p.Nm;
    u.j = u.szj % p.J;
    u.z = (u.szj / p.J) % p.Nz;
    u.s = u.szj / (p.J * p.Nz);
    return u;
}

template <class C>
__global__ void __launch_bounds__(2 * C::NT, 1) nl_rx_persist_kernel(const NlParams p, unsigned* chi_flag, unsigned epoch) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int NT = C::NT, NK = C::NK;
    const int grp = threadIdx.x / NT, tid = threadIdx.x - grp * NT;
    unsigned char* base = smem_raw + (size_t)grp * C::STAGE_BYTES;
    float2* S = reinterpret_cast<float2*>(base);
    float4* stage4 = reinterpret_cast<float4*>(base);
    float4* W4 = reinterpret_cast<float4*>(base + C::S_ELEMS * 8);
    float2* twx = reinterpret_cast<float2*>(smem_raw + 2 * (size_t)C::STAGE_BYTES);
    float* Tall = reinterpret_cast<float*>(twx + C::NX);        // T[j][l]
    float* Ti = Tall + 16 * 23;                                 // -Tinv[l][j]
    __shared__ unsigned long long stage_bar[2];
    __shared__ int last_flag[2];

    if (tid == 0) mbar_init(&stage_bar[grp], 1);
    for (int i = threadIdx.x; i < C::NX; i += 2 * NT) twx[i] = __ldg(p.twx + i);
    for (int i = threadIdx.x; i < p.Nl * p.J; i += 2 * NT) {
        Tall[i] = __ldg(p.T + i);
        Ti[i] = -__ldg(p.Tinv + i);                             // out = -N
    }
    __syncthreads();

    const int n_chi = p.Ns * p.Nz * p.J, n_items = n_chi + n_chi * p.Nm;
    const int G = gridDim.x * 2, gid = blockIdx.x * 2 + grp;
    const size_t lstride = (size_t)p.Nz * NK;
    unsigned bar_parity = 0;
    bool staged = false;            // chunk 0 of the current bracket unit has already been requested
    int pend_unit = -1;             // unit whose node plane is stored but not yet published

    auto request_chunk0 = [&](int unit) {      // thread 0 of the group
        const RxUnit u = rx_decode(unit, p);
        const float2* g0 = p.g + ((size_t)(u.s * p.Nm + u.m) * p.Nl * p.Nz + u.z) * NK;
        const int nl = min(C::CAP, p.Nl);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        mbar_expect_tx(&stage_bar[grp], (unsigned)(nl * NK * sizeof(float2)));
        for (int l = 0; l < nl; ++l) bulk_g2s(S + (size_t)l * NK, g0 + (size_t)l * lstride, NK * sizeof(float2), &stage_bar[grp]);
    };
    auto publish_pending = [&]() {             // one thread; the group barrier after the node-plane stores precedes it
        if (pend_unit >= 0 && tid == NT - 1) {
            const RxUnit u = rx_decode(pend_unit, p);
            __threadfence();        // release: stores -> barrier -> fence -> atomic
            atomicAdd(p.count + (u.s * p.Nm + u.m) * p.Nz + u.z, 1u);
        }
        pend_unit = -1;
    };
    // a8 as work items of their own: (s,m,z) number i belongs to group G-1 - (i mod G) (the groups with the fewest
    // bracket units come first), which forms out_l = - sum_j Tinv[l][j] Bhat_j once all J node planes have arrived.
    // Polled without blocking after every bracket unit -- the loads then share the wait for the next unit's
    // planes -- and with blocking once the group has published all its own units (so nobody can wait forever).
    const int n_smz = p.Ns * p.Nm * p.Nz;
    int lag_item = G - 1 - gid;
    auto laguerre_items = [&](bool block) {
        while (lag_item < n_smz) {
            if (tid == 0) {
                unsigned c = ld_acquire_u32(p.count + lag_item);
                while (block && c != (unsigned)p.J) { __nanosleep(200); c = ld_acquire_u32(p.count + lag_item); }
                last_flag[grp] = (c == (unsigned)p.J);
            }
            group_bar(grp, NT);
            const int ready = last_flag[grp];
            group_bar(grp, NT);                 // flag read by everyone before thread 0 may overwrite it
            if (!ready) break;
            const int z = lag_item % p.Nz, m = (lag_item / p.Nz) % p.Nm, sp = lag_item / (p.Nz * p.Nm);
            const float4* bh4 = reinterpret_cast<const float4*>(p.bhat + ((size_t)((sp * p.Nz + z) * p.J) * p.Nm + m) * NK);
            float4* out4 = reinterpret_cast<float4*>(p.out + (((size_t)(sp * p.Nm + m) * p.Nl) * p.Nz + z) * NK);
            rx_laguerre_inverse<C>(tid, CgPtr{bh4}, p.Nm * C::NK2, out4, (int)(lstride / 2), Ti, p.Nl, p.J);
            if (tid == 0) p.count[lag_item] = 0u;   // nobody touches this counter again before the next call
            lag_item += G;
        }
    };

    int round = -1;
    for (int item = gid; item < n_items; item += G) {
        ++round;
        GX_PHASE2(0);
        GX_PHASE2(1);
        if (item < n_chi) {
            // ---- a1 + a3 + a4 for the potential: chi plane (s,z,j)
            const int z = (item / p.J) % p.Nz;
            const float2* __restrict__ phi = p.phi + (size_t)(p.phi_by_unit ? item : z) * NK;
            const float* __restrict__ M = p.M + (size_t)(p.M_shared ? 0 : item) * NK;
            for (int i = tid; i < NK; i += NT) {
                const float2 f = __ldg(phi + i);
                const float mm = __ldg(M + i);
                S[i] = make_float2(f.x * mm, f.y * mm);
            }
            group_bar(grp, NT);
            rx_x_inverse_pass1<C>(tid, (const float2*)S, W4, (const float2*)twx, p.dkx, p.dky);
            group_bar(grp, NT);
            rx_x_inverse_pass2<C>(tid, W4);
            group_bar(grp, NT);
            rx_row_chi<C>(tid, (const float4*)W4, reinterpret_cast<float4*>(p.dchi) + (size_t)item * C::H * C::NX);
            group_bar(grp, NT);     // every thread's stores are ordered before thread 0's release below (cumulative)
            if (tid == 0) { __threadfence(); st_release_u32(chi_flag + item, epoch); }
            GX_PHASE2(2);
            continue;
        }
        const int unit = item - n_chi;
        const RxUnit u = rx_decode(unit, p);
        const float2* __restrict__ g0 = p.g + ((size_t)(u.s * p.Nm + u.m) * p.Nl * p.Nz + u.z) * NK;
        // ---- a2: forward Laguerre transform l -> node j, fused into the TMA-staged load
        if (!staged && tid == 0) request_chunk0(unit);
        staged = false;
        for (int l0 = 0; l0 < p.Nl;) {
            const bool first = l0 == 0;
            const int nl = min(first ? C::CAP : C::CAP - 1, p.Nl - l0);
            if (!first && tid == 0) {
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                mbar_expect_tx(&stage_bar[grp], (unsigned)(nl * NK * sizeof(float2)));
                for (int l = 0; l < nl; ++l)
                    bulk_g2s(S + (size_t)(l + 1) * NK, g0 + (size_t)(l0 + l) * lstride, NK * sizeof(float2), &stage_bar[grp]);
            }
            mbar_wait(&stage_bar[grp], bar_parity);
            bar_parity ^= 1u;
            rx_combine<C>(tid, stage4, Tall + u.j * p.Nl, l0, nl, first);
            group_bar(grp, NT);                                  // chunk consumed / S complete
            l0 += nl;
        }
        GX_PHASE2(3);
        publish_pending();          // previous unit: release fence + arrival atomic, in the warp with the least work below
        // ---- a3 + a4 (x part)
        rx_x_inverse_pass1<C>(tid, (const float2*)S, W4, (const float2*)twx, p.dkx, p.dky);
        group_bar(grp, NT);
        GX_PHASE2(4);
        rx_x_inverse_pass2<C>(tid, W4);
        GX_PHASE2(5);
        if (tid == 0) {             // this plane's chi pairs: ready flag of this call (set once, never waits later)
            while (ld_acquire_u32(chi_flag + u.szj) != epoch) __nanosleep(100);
        }
        group_bar(grp, NT);
        GX_PHASE2(6);
        // ---- a4 (y part) + a5 + a6 (y part) + a7 (ky)
        rx_row_bracket<C>(tid, W4, reinterpret_cast<const float4*>(p.dchi) + (size_t)u.szj * C::H * C::NX);
        group_bar(grp, NT);
        GX_PHASE2(7);
        // ---- a6 (x part) + a7 (kx)
        rx_x_forward_pass1<C>(tid, W4, (const float2*)twx);
        group_bar(grp, NT);
        rx_x_forward_pass2<C>(tid, (const float4*)W4, reinterpret_cast<float4*>(p.bhat + (size_t)unit * NK), p.scale);
        group_bar(grp, NT);         // plane buffer dead; every thread's node-plane stores precede thread 0's fence
        GX_PHASE2(8);
        // ---- the next unit's planes are requested at once; this unit is published (release: stores -> barrier
        // above -> fence -> atomic) during the next unit's x pass, see publish_pending
        const int next = item + G;
        if (tid == 0 && next < n_items) request_chunk0(next - n_chi);
        GX_PHASE2(9);
        staged = next < n_items;
        pend_unit = unit;
        laguerre_items(false);
        GX_PHASE2(10);
    }
    publish_pending();
    laguerre_items(true);
}

// ================================================================================================
// Warp-specialised software pipeline (family "rxw"): ONE persistent CTA per SM, 512 threads,
//     row workers  = warp groups 0-1 (192 of 256 threads used, 168 registers each after setmaxnreg.inc):
//                    y direction + bracket of item k (a4 y part, a5, a6 y part), chi rows, a8 items;
//     x workers    = warp groups 2-3 (256 threads, 88 registers after setmaxnreg.dec):
//                    staging + Laguerre combine + inverse x passes of item k+1, forward x passes of item k-1.
// Why (profiles/r02_rx_pipeline.md): with all warps walking the phases in lock step the FP32 pipe idles during
// the TMA wait, the latency-bound x passes and every barrier (48 % busy, 12.9 k cycles per unit and SM); the
// register file (168 registers for a 64-point row in one thread) allows no third lock-step group.  Shrinking
// the registers of the warps that never run the row phase pays for 8 more warps, and the two kinds of work
// overlap by construction: the row workers never wait for memory, the x workers hide their latencies behind
// the row phase.  Two plane buffers W4[2] alternate between the stages; hand-over is by named barriers
// (bar.arrive / bar.sync), the raw Laguerre planes of item k+1 are requested one stage ahead.
//
// Work list per CTA c: items c, c + grid, ... of [chi planes | bracket units]; chi items come first and never wait.
template <int N> __device__ __forceinline__ void reg_alloc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N> __device__ __forceinline__ void reg_dealloc() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }
__device__ __forceinline__ void nbar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void nbar_arrive(int id, int n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }

template <class C>
struct RxwLayout {
    static constexpr int NROW = C::NX;            // row workers in use (one per x row)
    static constexpr int NXW = 256;               // x workers
    static constexpr int NTHREADS = 512;
    static constexpr int W4_BYTES = C::W4_ELEMS * 16;
    static constexpr int CAPW_MAX = (232448 - 2 * W4_BYTES - C::NX * 8 - 2 * 16 * 23 * 4 - 64) / (C::NK * 8);
    static constexpr int CAPW = CAPW_MAX > 8 ? 8 : CAPW_MAX;   // raw-plane slots of the staging area (slot 0 is S)
    static constexpr int STAGE_BYTES = CAPW * C::NK * 8;
    static constexpr int SMEM = 2 * W4_BYTES + STAGE_BYTES + C::NX * 8 + 2 * 16 * 23 * 4;
    static_assert(NROW <= 256 && NROW % 32 == 0, "row workers live in warp groups 0-1");
    static_assert(CAPW >= 2, "two plane buffers and the staging area do not fit in shared memory");
};
// named barriers: 1, 2 = W4[b] holds the inverse x transform (x workers arrive, row workers wait);
// 3, 4 = W4[b] holds the forward data after the first forward x pass (row workers arrive, x workers wait);
// 5 = x workers among themselves; 6 = row workers among themselves
enum { RXW_BAR_INV = 1, RXW_BAR_FWD = 3, RXW_BAR_X = 5, RXW_BAR_ROW = 6 };

__device__ __forceinline__ void mbar_expect_tx_noarrive(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.expect_tx.relaxed.cta.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}

#ifdef GX_PHASE_TIMING
#define GX_PHASE3(i) do { if ((threadIdx.x == 256 || threadIdx.x == 0) && cid < 256 && k < 16) gx_phase2_clk[(cid * 16 + k) * 12 + (i)] = gx_globaltimer(); } while (0)
#else
#define GX_PHASE3(i) do { } while (0)
#endif
template <class C>
__global__ void __launch_bounds__(512, 1) nl_rx_pipeline_kernel(const NlParams p, unsigned* chi_flag, unsigned epoch) {
    using L = RxwLayout<C>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int NK = C::NK, NROW = L::NROW, NXW = L::NXW, NBOTH = NROW + NXW;
    float4* W4b[2] = {reinterpret_cast<float4*>(smem_raw), reinterpret_cast<float4*>(smem_raw + L::W4_BYTES)};
    unsigned char* stage = smem_raw + 2 * L::W4_BYTES;
    float2* S = reinterpret_cast<float2*>(stage);
    float4* stage4 = reinterpret_cast<float4*>(stage);
    float2* twx = reinterpret_cast<float2*>(stage + L::STAGE_BYTES);
    float* Tall = reinterpret_cast<float*>(twx + C::NX);        // T[j][l]
    float* Ti = Tall + 16 * 23;                                 // -Tinv[l][j]
    __shared__ unsigned long long stage_bar;
    __shared__ int row_flag;

    if (threadIdx.x == 0) mbar_init(&stage_bar, 1);
    for (int i = threadIdx.x; i < C::NX; i += L::NTHREADS) twx[i] = __ldg(p.twx + i);
    for (int i = threadIdx.x; i < p.Nl * p.J; i += L::NTHREADS) {
        Tall[i] = __ldg(p.T + i);
        Ti[i] = -__ldg(p.Tinv + i);                             // out = -N
    }
    __syncthreads();

    const int n_chi = p.Ns * p.Nz * p.J, n_items = n_chi + n_chi * p.Nm;
    const int G = gridDim.x, cid = blockIdx.x;
    const size_t lstride = (size_t)p.Nz * NK;

    if (threadIdx.x >= 256) {
        // ======================================================================== x workers
        reg_dealloc<88>();
        const int tid = threadIdx.x - 256;
        unsigned bar_parity = 0;
        const int nl0 = min(L::CAPW, p.Nl);                              // planes of the first staging chunk
        auto plane_src = [&](int unit, int l) {
            const RxUnit u = rx_decode(unit, p);
            return p.g + ((size_t)(u.s * p.Nm + u.m) * p.Nl * p.Nz + u.z) * NK + (size_t)l * lstride;
        };
        // first chunk in two steps: planes 1.. land in slots 1.. (free once the combine is done), plane 0 lands on S
        // (free once the first inverse x pass has read it); the arrive of step B completes the mbarrier phase
        auto request_upper = [&](int unit) {                            // one thread
            if (nl0 > 1) {
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                mbar_expect_tx_noarrive(&stage_bar, (unsigned)((nl0 - 1) * NK * sizeof(float2)));
                for (int l = 1; l < nl0; ++l) bulk_g2s(S + (size_t)l * NK, plane_src(unit, l), NK * sizeof(float2), &stage_bar);
            }
        };
        auto request_plane0 = [&](int unit) {                           // one thread
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            mbar_expect_tx(&stage_bar, (unsigned)(NK * sizeof(float2)));
            bulk_g2s(S, plane_src(unit, 0), NK * sizeof(float2), &stage_bar);
        };
        bool staged = false;
        int k = 0;
        for (int item = cid; item < n_items + G; item += G, ++k) {
            const int b = k & 1;
            const int next = item + G;
            const bool next_bracket = next < n_items && next >= n_chi;
            GX_PHASE3(0);
            if (item < n_items) {
                // ---- produce item k into W4[b]: compact plane S, then the inverse x passes
                if (item < n_chi) {
                    const int z = (item / p.J) % p.Nz;
                    const float2* __restrict__ phi = p.phi + (size_t)(p.phi_by_unit ? item : z) * NK;
                    const float* __restrict__ M = p.M + (size_t)(p.M_shared ? 0 : item) * NK;
                    for (int i = tid; i < NK; i += NXW) {
                        const float2 f = __ldg(phi + i);
                        const float mm = __ldg(M + i);
                        S[i] = make_float2(f.x * mm, f.y * mm);
                    }
                    nbar_sync(RXW_BAR_X, NXW);
                } else {
                    const int unit = item - n_chi;
                    const RxUnit u = rx_decode(unit, p);
                    if (!staged && tid == 0) { request_upper(unit); request_plane0(unit); }
                    staged = false;
                    for (int l0 = 0; l0 < p.Nl;) {
                        const bool first = l0 == 0;
                        const int nl = first ? nl0 : min(L::CAPW - 1, p.Nl - l0);
                        if (!first && tid == 0) {
                            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                            mbar_expect_tx(&stage_bar, (unsigned)(nl * NK * sizeof(float2)));
                            for (int l = 0; l < nl; ++l) bulk_g2s(S + (size_t)(l + 1) * NK, plane_src(unit, l0 + l), NK * sizeof(float2), &stage_bar);
                        }
                        mbar_wait(&stage_bar, bar_parity);
                        bar_parity ^= 1u;
                        GX_PHASE3(5);
                        rx_combine<C, NXW>(tid, stage4, Tall + u.j * p.Nl, l0, nl, first);
                        nbar_sync(RXW_BAR_X, NXW);                   // chunk consumed / S complete
                        l0 += nl;
                    }
                }
                if (next_bracket && tid == 0) request_upper(next - n_chi);      // slots 1.. are dead from here on
                GX_PHASE3(1);
                rx_x_inverse_pass1_single<C, NXW>(tid, (const float2*)S, W4b[b], (const float2*)twx, p.dkx, p.dky);
                nbar_sync(RXW_BAR_X, NXW);
                if (next_bracket) {                                              // S is dead from here on
                    if (tid == 0) request_plane0(next - n_chi);
                    staged = true;
                }
                rx_x_inverse_pass2_single<C, NXW>(tid, W4b[b]);
                __threadfence_block();
                nbar_arrive(RXW_BAR_INV + b, NBOTH);                 // W4[b] ready for the row workers
            }
            GX_PHASE3(2);
            // ---- retire item k-1 from W4[b^1]: second forward x pass of a bracket unit, then publish its node plane
            if (k >= 1) {
                const int prev = item - G;
                nbar_sync(RXW_BAR_FWD + (b ^ 1), NBOTH);             // rows + first forward x pass of item k-1 done
                GX_PHASE3(3);
                if (prev >= n_chi) {
                    const int unit = prev - n_chi;
                    rx_x_forward_pass2<C, NXW>(tid, (const float4*)W4b[b ^ 1], reinterpret_cast<float4*>(p.bhat + (size_t)unit * NK), p.scale);
                    nbar_sync(RXW_BAR_X, NXW);                       // node-plane stores precede the fence below (cumulative)
                    if (tid == NXW - 1) {
                        const RxUnit u = rx_decode(unit, p);
                        __threadfence();                             // release: stores -> barrier -> fence -> atomic
                        atomicAdd(p.count + (u.s * p.Nm + u.m) * p.Nz + u.z, 1u);
                    }
                }
                GX_PHASE3(4);
            }
        }
    } else {
        // ======================================================================== row workers
        reg_alloc<168>();
        const int tid = threadIdx.x;
        if (tid >= NROW) return;                                     // spare warps of warp group 1
        // a8 items: (s,m,z) number i belongs to CTA G-1 - (i mod G); polled after every item, blocking at the end
        const int n_smz = p.Ns * p.Nm * p.Nz;
        int lag_item = G - 1 - cid;
        auto laguerre_items = [&](bool block) {
            while (lag_item < n_smz) {
                if (tid == 0) {
                    unsigned c = ld_acquire_u32(p.count + lag_item);
                    while (block && c != (unsigned)p.J) { __nanosleep(200); c = ld_acquire_u32(p.count + lag_item); }
                    row_flag = (c == (unsigned)p.J);
                }
                nbar_sync(RXW_BAR_ROW, NROW);
                const int ready = row_flag;
                nbar_sync(RXW_BAR_ROW, NROW);
                if (!ready) break;
                const int z = lag_item % p.Nz, m = (lag_item / p.Nz) % p.Nm, sp = lag_item / (p.Nz * p.Nm);
                const float4* bh4 = reinterpret_cast<const float4*>(p.bhat + ((size_t)((sp * p.Nz + z) * p.J) * p.Nm + m) * NK);
                float4* out4 = reinterpret_cast<float4*>(p.out + (((size_t)(sp * p.Nm + m) * p.Nl) * p.Nz + z) * NK);
                rx_laguerre_inverse<C>(tid, CgPtr{bh4}, p.Nm * C::NK2, out4, (int)(lstride / 2), Ti, p.Nl, p.J);
                if (tid == 0) p.count[lag_item] = 0u;               // nobody touches this counter again before the next call
                lag_item += G;
            }
        };
        int k = 0;
        for (int item = cid; item < n_items; item += G, ++k) {
            const int b = k & 1;
            GX_PHASE3(6);
            nbar_sync(RXW_BAR_INV + b, NBOTH);                       // inverse x transform of item k is in W4[b]
            GX_PHASE3(7);
            if (item < n_chi) {
                rx_row_chi<C>(tid, (const float4*)W4b[b], reinterpret_cast<float4*>(p.dchi) + (size_t)item * C::H * C::NX);
                nbar_sync(RXW_BAR_ROW, NROW);                        // every thread's stores precede thread 0's release
                if (tid == 0) { __threadfence(); st_release_u32(chi_flag + item, epoch); }
            } else {
                const RxUnit u = rx_decode(item - n_chi, p);
                if (tid == 0) while (ld_acquire_u32(chi_flag + u.szj) != epoch) __nanosleep(100);
                nbar_sync(RXW_BAR_ROW, NROW);
                GX_PHASE3(8);
                rx_row_bracket<C>(tid, W4b[b], reinterpret_cast<const float4*>(p.dchi) + (size_t)u.szj * C::H * C::NX);
                nbar_sync(RXW_BAR_ROW, NROW);
                rx_x_forward_pass1<C>(tid, W4b[b], (const float2*)twx);      // a6 (x part), first pass: fits the row workers' slack
            }
            __threadfence_block();
            nbar_arrive(RXW_BAR_FWD + b, NBOTH);                     // W4[b] handed back to the x workers
            GX_PHASE3(9);
            laguerre_items(false);
            GX_PHASE3(10);
        }
        laguerre_items(true);
    }
}
#endif  // __CUDACC__

}  // namespace gx
