// nl_kernels.cuh -- sm_100a kernels of the nonlinear E×B term (App. D).
//
// One CTA evaluates one "unit": a (kx,ky) plane that stays in shared memory from the compact
// spectral input to the compact spectral output.  Steps (SURVEY.md / DESIGN.md rows a1-a8):
//
//   chi_planes_kernel   unit (s,z,j):    chi = M.Phi (a1) -> (i kx, i ky) (a3) -> inverse 2D FFT (a4)
//                                        -> real-space (d_x chi, d_y chi) pairs in the workspace
//   bracket_kernel      unit (s,m,z,j):  gt = sum_l T[j][l] G_l (a2) -> (i kx, i ky) (a3) -> inverse 2D FFT
//                                        (a4) -> bracket with the chi pairs (a5) -> forward 2D FFT (a6)
//                                        -> 2/3-rule truncation (a7) -> Bhat_j(k) in the workspace
//   laguerre_inverse_kernel  (s,m,z):    out_l = - sum_j Tinv[l][j] Bhat_j (a8)
//
// FFT design (differs from the paper's cuFFT calls):
//  * The two real fields d_x f and d_y f are transformed as ONE complex field
//    u = d_x f + i d_y f, whose spectrum over the reality-extended set is U(k) = (i kx - ky) f(k):
//    one complex 2D transform instead of two complex-to-real ones.  On the way back two x-rows of
//    the real bracket are packed as re/im of one complex row and separated after the y transform.
//  * Zero columns/rows of the 2/3-rule padding are never transformed: the x pass runs on the
//    2*naky-1 non-zero ky columns (inverse) / naky kept columns (forward).
//  * Each 1D transform is two register-radix passes (N = R1*R2, radices <= 16) over shared memory.
//    The inverse is decimation-in-time with in-place, digit-transposed output (position
//    k1*R2+k2 holds index k1+R1*k2); the forward is the matching decimation-in-frequency that reads
//    the transposed order and ends in natural order.  The real-space fields therefore live in a
//    permuted (x,y) order, which is harmless because the bracket is pointwise and the chi planes are
//    produced by the same code in the same order.  No bit/digit-reversal pass exists anywhere.
//  * The y transforms run on batches of RB x-rows through a scratch tile S[y][row]; lanes map to
//    rows, so every shared access is either contiguous or has the odd stride 2*naky-1.
#pragma once
#include "dft_regs.cuh"

namespace gx {

template <int NX_, int NY_, int RX1_, int RX2_, int RY1_, int RY2_, int RB_, int NT_, int MINB_, bool STAGE_>
struct PlaneCfg {
    static constexpr int NX = NX_, NY = NY_, RX1 = RX1_, RX2 = RX2_, RY1 = RY1_, RY2 = RY2_;
    static constexpr int RB = RB_, NT = NT_, MINB = MINB_;
    static constexpr bool STAGE = STAGE_;
    static constexpr int K = (NX - 1) / 3, Q = (NY - 1) / 3;
    static constexpr int NAKX = 2 * K + 1, NAKY = Q + 1, NCOL = 2 * Q + 1, NK = NAKX * NAKY;
    static constexpr int HB = RB / 2, NBATCH = NX / RB;
    static constexpr int W_ELEMS = NX * NCOL;
    static constexpr int S_ELEMS = (STAGE && NK > NY * RB) ? NK : NY * RB;
    static constexpr int SMEM_BYTES = (W_ELEMS + S_ELEMS + NX + NY) * (int)sizeof(float2);
    static_assert(RX1 * RX2 == NX && RY1 * RY2 == NY, "radix split");
    static_assert(NX % RB == 0 && RB % 2 == 0 && NX % 2 == 0, "row batches");
    static_assert(SMEM_BYTES <= 232448, "plane does not fit in shared memory");
};

struct NlParams {
    const float2* g;      // [s][m][l][z][kx][ky]
    const float2* phi;    // [z][kx][ky]
    float2* dchi;         // [s][z][j][py][px]  (d_x chi, d_y chi), permuted real-space order
    float2* bhat;         // [s][z][j][m][kx][ky]
    float2* out;          // [s][m][l][z][kx][ky]
    const float* M;       // [s][z][j][kx][ky]
    const float* T;       // [j][l]
    const float* Tinv;    // [l][j]
    const float2* twx;    // e^{+2 pi i t/NX}
    const float2* twy;
    float dkx, dky, scale;
    int Nz, Nl, Nm, Ns, J;
};

// ------------------------------------------------------------------------------------------------
// inverse x transform of U(k) = (i kx - ky) f(k) on the 2*naky-1 non-zero columns.
// fetch(i, q): compact f at kx row i, ky column q >= 0.
template <class C, class Fetch>
__device__ __forceinline__ void x_inverse(float2* __restrict__ W, const float2* __restrict__ twx,
                                          float dkx, float dky, Fetch fetch) {
    constexpr int NX = C::NX, K = C::K, NCOL = C::NCOL, NAKY = C::NAKY, NAKX = C::NAKX;
    constexpr int R1 = C::RX1, R2 = C::RX2;
    // pass 1: for each (n2, column): DFT_R1 over n1 of input n = n1*R2+n2, twiddle, in-place slot
    for (int t = threadIdx.x; t < R2 * NCOL; t += C::NT) {
        const int n2 = t / NCOL, c = t - n2 * NCOL;
        const int q = c < NAKY ? c : c - NCOL;
        const int qa = q < 0 ? -q : q;
        const float kyq = dky * (float)q;
        float2 v[R1];
#pragma unroll
        for (int n1 = 0; n1 < R1; ++n1) {
            const int n = n1 * R2 + n2;
            v[n1] = make_float2(0.f, 0.f);
            if (n1 * R2 <= K || n1 * R2 + R2 - 1 >= NX - K) {        // compile-time prune of all-zero n1
                int a = 0;
                bool nz = false;
                if (n <= K) { a = n; nz = true; }
                else if (n >= NX - K) { a = n - NX; nz = true; }
                if (nz) {
                    const int as = q >= 0 ? a : -a;
                    const int i = as >= 0 ? as : as + NAKX;
                    float2 f = fetch(i, qa);
                    if (q < 0) f.y = -f.y;
                    const float kxa = dkx * (float)a;
                    v[n1] = make_float2(-kyq * f.x - kxa * f.y, kxa * f.x - kyq * f.y);
                }
            }
        }
        dft<R1, +1>(v);
#pragma unroll
        for (int k1 = 0; k1 < R1; ++k1)
            W[(k1 * R2 + n2) * NCOL + c] = k1 == 0 ? v[0] : cmul(v[k1], twx[n2 * k1]);
    }
    __syncthreads();
    // pass 2: for each (k1, column): DFT_R2 over n2; position k1*R2+k2 <- x = k1 + R1*k2
    for (int t = threadIdx.x; t < R1 * NCOL; t += C::NT) {
        const int k1 = t / NCOL, c = t - k1 * NCOL;
        float2 v[R2];
#pragma unroll
        for (int n2 = 0; n2 < R2; ++n2) v[n2] = W[(k1 * R2 + n2) * NCOL + c];
        dft<R2, +1>(v);
#pragma unroll
        for (int k2 = 0; k2 < R2; ++k2) W[(k1 * R2 + k2) * NCOL + c] = v[k2];
    }
    __syncthreads();
}

// y inverse pass 1 for a batch of RB rows: W rows (2*naky-1 non-zero inputs) -> S[(k1*RY2+n2)*RB + r]
template <class C, bool PAIRED>
__device__ __forceinline__ void y_inverse_pass1(const float2* __restrict__ W, float2* __restrict__ S,
                                                const float2* __restrict__ twy, int bt) {
    constexpr int NX = C::NX, NY = C::NY, Q = C::Q, NCOL = C::NCOL, RB = C::RB, HB = C::HB;
    constexpr int R1 = C::RY1, R2 = C::RY2;
    for (int t = threadIdx.x; t < R2 * RB; t += C::NT) {
        const int n2 = t / RB, r = t - n2 * RB;
        const int row = PAIRED ? (r < HB ? bt * HB + r : bt * HB + (r - HB) + NX / 2) : bt * RB + r;
        const float2* __restrict__ Wr = W + row * NCOL;
        float2 v[R1];
#pragma unroll
        for (int n1 = 0; n1 < R1; ++n1) {
            const int n = n1 * R2 + n2;
            v[n1] = make_float2(0.f, 0.f);
            if (n1 * R2 <= Q || n1 * R2 + R2 - 1 >= NY - Q) {
                if (n <= Q) v[n1] = Wr[n];
                else if (n >= NY - Q) v[n1] = Wr[n - NY + NCOL];
            }
        }
        dft<R1, +1>(v);
#pragma unroll
        for (int k1 = 0; k1 < R1; ++k1)
            S[(k1 * R2 + n2) * RB + r] = k1 == 0 ? v[0] : cmul(v[k1], twy[n2 * k1]);
    }
    __syncthreads();
}

// forward x transform on the naky kept columns; W holds Bhat(x, q) at permuted x positions.
// Writes the 2K+1 kept kx rows (compact order) times `scale` to out[i*NAKY + q].
template <class C>
__device__ __forceinline__ void x_forward(float2* __restrict__ W, const float2* __restrict__ twx,
                                          float2* __restrict__ out, float scale) {
    constexpr int NX = C::NX, K = C::K, NCOL = C::NCOL, NAKY = C::NAKY, NAKX = C::NAKX;
    constexpr int R1 = C::RX1, R2 = C::RX2;
    for (int t = threadIdx.x; t < R1 * NAKY; t += C::NT) {
        const int a = t / NAKY, q = t - a * NAKY;
        float2 v[R2];
#pragma unroll
        for (int b = 0; b < R2; ++b) v[b] = W[(a * R2 + b) * NCOL + q];
        dft<R2, -1>(v);
#pragma unroll
        for (int d = 0; d < R2; ++d)
            W[(a * R2 + d) * NCOL + q] = d == 0 ? v[0] : cmul_conj(v[d], twx[a * d]);
    }
    __syncthreads();
    for (int t = threadIdx.x; t < R2 * NAKY; t += C::NT) {
        const int d = t / NAKY, q = t - d * NAKY;
        float2 v[R1];
#pragma unroll
        for (int a = 0; a < R1; ++a) v[a] = W[(a * R2 + d) * NCOL + q];
        dft<R1, -1>(v);
#pragma unroll
        for (int cc = 0; cc < R1; ++cc) {
            if (cc * R2 <= K || cc * R2 + R2 - 1 >= NX - K) {
                const int n = d + R2 * cc;
                int i = -1;
                if (n <= K) i = n;
                else if (n >= NX - K) i = n - NX + NAKX;
                if (i >= 0) out[i * NAKY + q] = make_float2(v[cc].x * scale, v[cc].y * scale);
            }
        }
    }
}

template <class C>
__device__ __forceinline__ void load_twiddles(float2* twx_s, float2* twy_s, const NlParams& p) {
    for (int i = threadIdx.x; i < C::NX; i += C::NT) twx_s[i] = p.twx[i];
    for (int i = threadIdx.x; i < C::NY; i += C::NT) twy_s[i] = p.twy[i];
}

// ================================================================================================
// a1 + a3 + a4 for the potential: real-space (d_x chi, d_y chi) of chi_{s,z,j} = M_{s,z,j} Phi_z.
template <class C>
__global__ void __launch_bounds__(C::NT, C::MINB) chi_planes_kernel(const NlParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2* W = reinterpret_cast<float2*>(smem_raw);
    float2* S = W + C::W_ELEMS;
    float2* twx = S + C::S_ELEMS;
    float2* twy = twx + C::NX;
    const int unit = blockIdx.x;                 // (s*Nz + z)*J + j
    const int z = (unit / p.J) % p.Nz;
    const float2* __restrict__ phi = p.phi + (size_t)z * C::NK;
    const float* __restrict__ M = p.M + (size_t)unit * C::NK;
    load_twiddles<C>(twx, twy, p);
    if constexpr (C::STAGE) {
        for (int i = threadIdx.x; i < C::NK; i += C::NT) {
            const float2 f = phi[i];
            const float m = M[i];
            S[i] = make_float2(f.x * m, f.y * m);
        }
        __syncthreads();
        x_inverse<C>(W, twx, p.dkx, p.dky, [&](int i, int q) { return S[i * C::NAKY + q]; });
    } else {
        __syncthreads();
        x_inverse<C>(W, twx, p.dkx, p.dky, [&](int i, int q) {
            const float2 f = __ldg(phi + i * C::NAKY + q);
            const float m = __ldg(M + i * C::NAKY + q);
            return make_float2(f.x * m, f.y * m);
        });
    }
    float2* __restrict__ dchi = p.dchi + (size_t)unit * C::NX * C::NY;
    constexpr int R1 = C::RY1, R2 = C::RY2, RB = C::RB;
    for (int bt = 0; bt < C::NBATCH; ++bt) {
        y_inverse_pass1<C, false>(W, S, twy, bt);
        for (int t = threadIdx.x; t < R1 * RB; t += C::NT) {
            const int k1 = t / RB, r = t - k1 * RB;
            float2 v[R2];
#pragma unroll
            for (int n2 = 0; n2 < R2; ++n2) v[n2] = S[(k1 * R2 + n2) * RB + r];
            dft<R2, +1>(v);
#pragma unroll
            for (int k2 = 0; k2 < R2; ++k2) dchi[(size_t)(k1 * R2 + k2) * C::NX + bt * RB + r] = v[k2];
        }
        __syncthreads();
    }
}

// ================================================================================================
// a2-a7 for one (s,m,z,j): Bhat_j(k) = F_k[ d_y chi d_x gt - d_x chi d_y gt ], 2/3-rule truncated.
template <class C>
__global__ void __launch_bounds__(C::NT, C::MINB) bracket_kernel(const NlParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2* W = reinterpret_cast<float2*>(smem_raw);
    float2* S = W + C::W_ELEMS;
    float2* twx = S + C::S_ELEMS;
    float2* twy = twx + C::NX;
    constexpr int NX = C::NX, NY = C::NY, Q = C::Q, NCOL = C::NCOL, RB = C::RB, HB = C::HB, NK = C::NK;
    constexpr int R1 = C::RY1, R2 = C::RY2;

    const int unit = blockIdx.x;                 // ((s*Nz + z)*J + j)*Nm + m
    const int m = unit % p.Nm;
    const int szj = unit / p.Nm;
    const int j = szj % p.J;
    const int z = (szj / p.J) % p.Nz;
    const int s = szj / (p.J * p.Nz);
    const size_t lstride = (size_t)p.Nz * NK;
    const float2* __restrict__ g0 = p.g + ((size_t)(s * p.Nm + m) * p.Nl * p.Nz + z) * NK;
    const float* __restrict__ Tj = p.T + j * p.Nl;

    load_twiddles<C>(twx, twy, p);
    // ---- a2: forward Laguerre transform l -> node j, fused into the load
    if constexpr (C::STAGE) {
        for (int i = threadIdx.x; i < NK; i += C::NT) {
            float2 acc = make_float2(0.f, 0.f);
            for (int l = 0; l < p.Nl; ++l) {
                const float tl = __ldg(Tj + l);
                const float2 f = g0[(size_t)l * lstride + i];
                acc.x = fmaf(tl, f.x, acc.x);
                acc.y = fmaf(tl, f.y, acc.y);
            }
            S[i] = acc;
        }
        __syncthreads();
        x_inverse<C>(W, twx, p.dkx, p.dky, [&](int i, int q) { return S[i * C::NAKY + q]; });
    } else {
        __syncthreads();
        const int Nl = p.Nl;
        x_inverse<C>(W, twx, p.dkx, p.dky, [&](int i, int q) {
            float2 acc = make_float2(0.f, 0.f);
            for (int l = 0; l < Nl; ++l) {
                const float tl = __ldg(Tj + l);
                const float2 f = __ldg(g0 + (size_t)l * lstride + i * C::NAKY + q);
                acc.x = fmaf(tl, f.x, acc.x);
                acc.y = fmaf(tl, f.y, acc.y);
            }
            return acc;
        });
    }

    const float2* __restrict__ dchi = p.dchi + (size_t)szj * NX * NY;
    for (int bt = 0; bt < C::NBATCH; ++bt) {
        // ---- a4 (y part): rows p and p+NX/2 of the batch
        y_inverse_pass1<C, true>(W, S, twy, bt);
        // ---- a4 (last pass) + a5 bracket + a6 (first forward pass), all in registers
        for (int t = threadIdx.x; t < R1 * HB; t += C::NT) {
            const int k1 = t / HB, rp = t - k1 * HB;
            float2 c[R2];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int r = rp + h * HB;
                const int row = bt * HB + rp + h * (NX / 2);
                float2 v[R2];
#pragma unroll
                for (int n2 = 0; n2 < R2; ++n2) v[n2] = S[(k1 * R2 + n2) * RB + r];
                dft<R2, +1>(v);
#pragma unroll
                for (int k2 = 0; k2 < R2; ++k2) {
                    const float2 d = __ldg(dchi + (size_t)(k1 * R2 + k2) * NX + row);
                    const float b = fmaf(d.y, v[k2].x, -d.x * v[k2].y);   // d_y chi d_x g - d_x chi d_y g
                    if (h == 0) c[k2].x = b; else c[k2].y = b;
                }
            }
            dft<R2, -1>(c);
#pragma unroll
            for (int d = 0; d < R2; ++d)
                S[(k1 * R2 + d) * RB + rp] = d == 0 ? c[0] : cmul_conj(c[d], twy[k1 * d]);
        }
        __syncthreads();
        // ---- a6 (last y pass) + a7 (keep ky <= Q) + separation of the packed row pair
        for (int t = threadIdx.x; t < (R2 / 2 + 1) * HB; t += C::NT) {
            const int dd = t / HB, rp = t - dd * HB;
            const int d0 = dd, d1 = (R2 - dd) % R2;
            float2 u0[R1], u1[R1];
#pragma unroll
            for (int a = 0; a < R1; ++a) u0[a] = S[(a * R2 + d0) * RB + rp];
            dft<R1, -1>(u0);
            if (d1 != d0) {
#pragma unroll
                for (int a = 0; a < R1; ++a) u1[a] = S[(a * R2 + d1) * RB + rp];
                dft<R1, -1>(u1);
            } else {
#pragma unroll
                for (int a = 0; a < R1; ++a) u1[a] = u0[a];
            }
            float2* __restrict__ W0 = W + (bt * HB + rp) * NCOL;
            float2* __restrict__ W1 = W0 + (NX / 2) * NCOL;
#pragma unroll
            for (int cc = 0; cc <= Q / R2; ++cc) {
                // class d0: k = d0 + R2*cc, partner NY-k in class d1
                {
                    const int k = d0 + R2 * cc;
                    if (k <= Q) {
                        const float2 A = u0[cc];
                        const float2 B = (d0 == 0) ? u1[(R1 - cc) % R1] : u1[R1 - 1 - cc];
                        W0[k] = make_float2(0.5f * (A.x + B.x), 0.5f * (A.y - B.y));
                        W1[k] = make_float2(0.5f * (A.y + B.y), 0.5f * (B.x - A.x));
                    }
                }
                if (d1 != d0) {
                    const int k = d1 + R2 * cc;
                    if (k <= Q) {
                        const float2 A = u1[cc];
                        const float2 B = u0[R1 - 1 - cc];
                        W0[k] = make_float2(0.5f * (A.x + B.x), 0.5f * (A.y - B.y));
                        W1[k] = make_float2(0.5f * (A.y + B.y), 0.5f * (B.x - A.x));
                    }
                }
            }
        }
        __syncthreads();
    }
    // ---- a6 (x part) + a7 (keep |kx| <= K)
    x_forward<C>(W, twx, p.bhat + (size_t)unit * NK, p.scale);
}

// ================================================================================================
// a8: out[s,m,l,z,k] = - sum_j Tinv[l][j] Bhat[s,z,j,m,k]
template <int MAXL, int MAXJ>
__global__ void __launch_bounds__(256) laguerre_inverse_kernel(const NlParams p, int nk) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    const int smz = blockIdx.y;                   // (s*Nm + m)*Nz + z
    const int z = smz % p.Nz;
    const int m = (smz / p.Nz) % p.Nm;
    const int s = smz / (p.Nz * p.Nm);
    __shared__ float Ti[MAXL * MAXJ];
    for (int i = threadIdx.x; i < p.Nl * p.J; i += blockDim.x) Ti[i] = p.Tinv[i];
    __syncthreads();
    if (k >= nk) return;
    float2 b[MAXJ];
#pragma unroll
    for (int j = 0; j < MAXJ; ++j)
        if (j < p.J) b[j] = p.bhat[((size_t)((s * p.Nz + z) * p.J + j) * p.Nm + m) * nk + k];
#pragma unroll
    for (int l = 0; l < MAXL; ++l) {
        if (l < p.Nl) {
            float2 acc = make_float2(0.f, 0.f);
#pragma unroll
            for (int j = 0; j < MAXJ; ++j)
                if (j < p.J) {
                    const float t = Ti[l * p.J + j];
                    acc.x = fmaf(-t, b[j].x, acc.x);
                    acc.y = fmaf(-t, b[j].y, acc.y);
                }
            p.out[(((size_t)(s * p.Nm + m) * p.Nl + l) * p.Nz + z) * nk + k] = acc;
        }
    }
}

}  // namespace gx
