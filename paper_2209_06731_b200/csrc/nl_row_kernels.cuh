// nl_row_kernels.cuh -- "row" kernel family of the nonlinear E×B term for NY = 64 (sm_100a, fp32).
// PAPER.md lines 646-655 (App. D Eq. D1 line 1); rows a1-a7 of SURVEY.md section 8(a).
//
// The r01b captures (profiles/r01b_bracket_families_ncu_full.md) show that the block-synchronous kernels are
// bound by the shared-memory/LSU data pipe and by CTA barriers, not by instruction issue.  This family keeps
// the x passes of nl_kernels.cuh (two register-radix passes over the W plane in shared memory) but does the
// whole y direction of one x row inside ONE thread, in registers:
//     43 non-zero ky inputs of the row  ->  64-point inverse transform (8 x 8, compile-time twiddles and zero
//     masks)  ->  bracket with the chi pairs at the row's 64 y points  ->  64-point REAL forward transform
//     (32-point complex transform of the even/odd packing + split)  ->  22 kept ky outputs back into the row.
// Nothing of the y direction touches shared memory (no S tile, no twiddle table, no per-batch barriers):
// per unit the kernel issues about half the shared-memory wavefronts of the two-pass families and 7
// instead of 14 CTA barriers.  One thread per x row: 192 threads per CTA for the Cyclone plane, two CTAs
// per SM, <= 168 registers per thread.
//
// Real space is in natural y order and digit-permuted x order (the x passes leave rows permuted; harmless,
// see nl_kernels.cuh).  Workspace dchi for this family: float2 (d_x chi, d_y chi) at [y][x position].
#pragma once
#include "nl_kernels.cuh"

namespace gx {

template <int NX_, int NY_, int RX1_, int RX2_, int NT_, int MINB_>
struct RowCfg {
    static constexpr int NX = NX_, NY = NY_, RX1 = RX1_, RX2 = RX2_, NT = NT_, MINB = MINB_;
    static constexpr int K = (NX - 1) / 3, Q = (NY - 1) / 3;
    static constexpr int NAKX = 2 * K + 1, NAKY = Q + 1, NCOL = 2 * Q + 1, NK = NAKX * NAKY;
    static constexpr int W_ELEMS = NX * NCOL;
    // compact plane after the Laguerre combine; padded so that W + S hold 4 raw planes for the TMA staging
    static constexpr int S_MIN = 4 * NK > W_ELEMS ? 4 * NK - W_ELEMS : 0;
    static constexpr int S_ELEMS = ((NK > S_MIN ? NK : S_MIN) + 1) / 2 * 2;
    static constexpr int SMEM_BYTES = (W_ELEMS + S_ELEMS + NX) * (int)sizeof(float2);
    static constexpr bool STAGE = true;
    static constexpr unsigned zero_mask(int R1, int R2, int N, int KK) {
        unsigned m = 0;
        for (int n1 = 0; n1 < R1; ++n1)
            if (!(n1 * R2 <= KK || n1 * R2 + R2 - 1 >= N - KK)) m |= 1u << n1;
        return m;
    }
    static constexpr unsigned ZMX = zero_mask(RX1, RX2, NX, K);
    static constexpr zm_t zero_mask_y() {
        zm_t m = 0;
        for (int n = 0; n < NY; ++n)
            if (n > Q && n < NY - Q) m |= 1ull << n;
        return m;
    }
    static constexpr zm_t ZMY = zero_mask_y();
    static_assert(NY == 64, "the single-thread y transform is written for 64 points");
    static_assert(RX1 * RX2 == NX && NK % 2 == 0, "radix split / 16-byte planes");
    static_assert(SMEM_BYTES <= 232448, "plane does not fit in shared memory");
};

// 64-point inverse transform of one W row (zero-padded 2/3-rule spectrum): v[y] = d_x f + i d_y f at y.
template <class C>
__device__ __forceinline__ void row_inverse(const float2* __restrict__ Wr, float2 (&v)[64]) {
    constexpr int NY = C::NY, Q = C::Q, NCOL = C::NCOL;
#pragma unroll
    for (int n = 0; n < NY; ++n) {
        if (n <= Q) v[n] = Wr[n];
        else if (n >= NY - Q) v[n] = Wr[n - NY + NCOL];
        else v[n] = make_float2(0.f, 0.f);
    }
    dft<64, +1, C::ZMY>(v);
}

// 64-point forward transform of the real sequence b -> the Q+1 kept coefficients into Wr[0..Q].
template <class C>
__device__ __forceinline__ void row_forward_real(float2* __restrict__ Wr, const float (&b)[64]) {
    constexpr int Q = C::Q;
    float2 z[32];
#pragma unroll
    for (int i = 0; i < 32; ++i) z[i] = make_float2(b[2 * i], b[2 * i + 1]);
    dft<32, -1>(z);
#pragma unroll
    for (int k = 0; k <= Q; ++k) {
        const float2 a = z[k], c = z[(32 - k) % 32];
        // E = (Z[k] + conj Z[32-k])/2 (even samples), O = (Z[k] - conj Z[32-k])/(2i) (odd samples)
        const float2 e = make_float2(0.5f * (a.x + c.x), 0.5f * (a.y - c.y));
        const float2 o = make_float2(0.5f * (a.y + c.y), 0.5f * (c.x - a.x));
        Wr[k] = cadd(e, twiddle<64, -1>(o, k));
    }
}

// ================================================================================================
// a1 + a3 + a4 for the potential: real-space (d_x chi, d_y chi) of chi_{s,z,j} = M_{s,z,j} Phi_z.
template <class C>
__global__ void __launch_bounds__(C::NT, C::MINB) chi_planes_row_kernel(const NlParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2* W = reinterpret_cast<float2*>(smem_raw);
    float2* S = W + C::W_ELEMS;
    float2* twx = S + C::S_ELEMS;
    const int unit = blockIdx.x;                 // (s*Nz + z)*J + j
    const int z = (unit / p.J) % p.Nz;
    const float2* __restrict__ phi = p.phi + (size_t)(p.phi_by_unit ? unit : z) * C::NK;
    const float* __restrict__ M = p.M + (size_t)(p.M_shared ? 0 : unit) * C::NK;
    pdl_launch_dependents();
    for (int i = threadIdx.x; i < C::NX; i += C::NT) twx[i] = p.twx[i];
    for (int i = threadIdx.x; i < C::NK; i += C::NT) {
        const float2 f = __ldg(phi + i);
        const float m = __ldg(M + i);
        S[i] = make_float2(f.x * m, f.y * m);
    }
    __syncthreads();
    x_inverse<C, false>(W, twx, p.dkx, p.dky, S);
    float2* __restrict__ dchi = p.dchi + (size_t)unit * C::NX * C::NY;
    for (int row = threadIdx.x; row < C::NX; row += C::NT) {
        float2 v[64];
        row_inverse<C>(W + row * C::NCOL, v);
#pragma unroll
        for (int y = 0; y < 64; ++y) dchi[y * C::NX + row] = v[y];
    }
}

// ================================================================================================
// a2-a7 for one (s,m,z,j): Bhat_j(k) = F_k[ d_y chi d_x gt - d_x chi d_y gt ], 2/3-rule truncated.
template <class C>
__global__ void __launch_bounds__(C::NT, C::MINB) bracket_row_kernel(const NlParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2* W = reinterpret_cast<float2*>(smem_raw);
    float2* S = W + C::W_ELEMS;
    float2* twx = S + C::S_ELEMS;
    constexpr int NX = C::NX, NY = C::NY, NK = C::NK;

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
    for (int i = threadIdx.x; i < NX; i += C::NT) twx[i] = p.twx[i];
    // ---- a2: forward Laguerre transform l -> node j, fused into the TMA-staged load
    stage_combine_tma<C>(W, S, &stage_bar, bar_parity, g0, lstride, Tsh, p.Nl);
    __syncthreads();
    GX_PHASE(1);
    // ---- a3 + a4 (x part)
    x_inverse<C, false>(W, twx, p.dkx, p.dky, S);
    GX_PHASE(2);

    const float2* dchi = p.dchi + (size_t)szj * NX * NY;
    pdl_wait();                     // chi planes of this call are complete and visible from here on
    GX_PHASE(3);
    // ---- a4 (y part) + a5 + a6 (y part) + a7 (ky), one x row per thread, all in registers
    for (int row = threadIdx.x; row < NX; row += C::NT) {
        float2* __restrict__ Wr = W + row * C::NCOL;
        const float2* dc = dchi + row;     // written by the chi grid that overlaps this one (PDL): coherent loads after pdl_wait
        // chi pairs of the first output group are requested before the transform starts, those of group
        // k1+1 while group k1 is transformed: the L2 latency of dchi hides behind the butterflies
        float2 d[8], dn[8];
#pragma unroll
        for (int k2 = 0; k2 < 8; ++k2) d[k2] = dc[(8 * k2) * NX];
#pragma unroll
        for (int k2 = 0; k2 < 8; ++k2) {       // groups 1 and 2 towards L1 (no registers held)
            asm volatile("prefetch.global.L1 [%0];" ::"l"(dc + (1 + 8 * k2) * NX));
            asm volatile("prefetch.global.L1 [%0];" ::"l"(dc + (2 + 8 * k2) * NX));
        }
        float2 y[64];
        {
            float2 v[64];
#pragma unroll
            for (int n = 0; n < NY; ++n) {
                if (n <= C::Q) v[n] = Wr[n];
                else if (n >= NY - C::Q) v[n] = Wr[n - NY + C::NCOL];
                else v[n] = make_float2(0.f, 0.f);
            }
            dft_split_col<64, 8, 8, +1, C::ZMY, 0>(v, y);      // first stage over n1 + twiddles
        }
        float b[64];
#pragma unroll
        for (int k1 = 0; k1 < 8; ++k1) {
            if (k1 < 7) {
#pragma unroll
                for (int k2 = 0; k2 < 8; ++k2) dn[k2] = dc[(k1 + 1 + 8 * k2) * NX];
            }
            if (k1 < 5) {
#pragma unroll
                for (int k2 = 0; k2 < 8; ++k2) asm volatile("prefetch.global.L1 [%0];" ::"l"(dc + (k1 + 3 + 8 * k2) * NX));
            }
            float2 u[8];
#pragma unroll
            for (int n2 = 0; n2 < 8; ++n2) u[n2] = y[k1 * 8 + n2];
            Dft<8, +1, sub_mask_second<8, 8, C::ZMY>()>::run(u);
#pragma unroll
            for (int k2 = 0; k2 < 8; ++k2) {
                b[k1 + 8 * k2] = fmaf(d[k2].y, u[k2].x, -d[k2].x * u[k2].y);   // d_y chi d_x g - d_x chi d_y g
                d[k2] = dn[k2];
            }
        }
        row_forward_real<C>(Wr, b);
    }
    __syncthreads();
    GX_PHASE(4);
    // ---- a6 (x part) + a7 (keep |kx| <= K)
    x_forward<C>(W, twx, p.bhat + (size_t)unit * NK, p.scale);

    // ---- publish (see bracket_kernel)
    __syncthreads();
    GX_PHASE(5);
    if (threadIdx.x == 0) { __threadfence(); atomicAdd(p.count + (s * p.Nm + m) * p.Nz + z, 1u); }
}

}  // namespace gx
