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
//   laguerre_inverse_kernel  (s,m,z):    out_l = - sum_j Tinv[l][j] Bhat_j (a8), overlapping the bracket tail
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
#include <type_traits>

#include "dft_regs.cuh"

namespace gx {

// Optional phase timing (development builds only, -DGX_PHASE_TIMING): thread 0 of the first CTAs records
// clock64() at phase boundaries; read back with gx_debug_phase_clocks().
#ifdef GX_PHASE_TIMING
static __device__ long long gx_phase_clk[64 * 32];   // one copy per translation unit (development builds only)
#define GX_PHASE(i) do { if (threadIdx.x == 0 && blockIdx.x < 64) gx_phase_clk[blockIdx.x * 32 + (i)] = clock64(); } while (0)
#else
#define GX_PHASE(i) do { } while (0)
#endif


template <int NX_, int NY_, int RX1_, int RX2_, int RY1_, int RY2_, int RB_, int NT_, int MINB_, bool STAGE_>
struct PlaneCfg {
    static constexpr int NX = NX_, NY = NY_, RX1 = RX1_, RX2 = RX2_, RY1 = RY1_, RY2 = RY2_;
    static constexpr int RB = RB_, NT = NT_, MINB = MINB_;
    static constexpr bool STAGE = STAGE_;
    static constexpr int K = (NX - 1) / 3, Q = (NY - 1) / 3;
    static constexpr int NAKX = 2 * K + 1, NAKY = Q + 1, NCOL = 2 * Q + 1, NK = NAKX * NAKY;
    static constexpr int NKP = NK;               // elements of a compact plane in memory (differs from NK in transposed row configs)
    static constexpr bool TR = false;
    static constexpr int HB = RB / 2, NBATCH = NX / RB;
    // Which two x rows share one complex forward y transform: rows p and p + NX/2 (lanes of a half-warp then read rows
    // NX/2 apart, which lie in the same shared-memory banks whenever HB < 16: 26 % of the stellarator kernel's
    // wavefronts were conflicts) or, for the small batches, the adjacent rows 2p and 2p + 1 (conflict-free for HB <= 8).
    static constexpr bool ADJ = RB <= 16;
    // Position of (y = a*RY2 + b, row slot r) in the batch buffer S.  With batches of 16 rows the pair phases run 8 lanes
    // per y value and 4 values of a (2 KB apart) or of b (128 B apart) per warp, all in the same half of the banks
    // (25 % of the stellarator kernel's shared-memory wavefronts were conflicts): rows with odd a + b hold their two
    // halves swapped.
    static constexpr bool SWZ = RB == 16;
    __device__ __forceinline__ static int sidx(int a, int b, int r) {
        return (a * RY2 + b) * RB + (SWZ ? (r ^ (((a ^ b) & 1) * HB)) : r);
    }
    static constexpr int W_ELEMS = NX * NCOL;
    static constexpr int S_ELEMS = (STAGE && NK > NY * RB) ? NK : NY * RB;
    static constexpr int SMEM_BYTES = (W_ELEMS + S_ELEMS + NX + NY) * (int)sizeof(float2);
    // compile-time zero masks of the first inverse passes: input n = n1*R2 + n2 is padding for every n2
    static constexpr unsigned zero_mask(int R1, int R2, int N, int KK) {
        unsigned m = 0;
        for (int n1 = 0; n1 < R1; ++n1)
            if (!(n1 * R2 <= KK || n1 * R2 + R2 - 1 >= N - KK)) m |= 1u << n1;
        return m;
    }
    static constexpr unsigned ZMX = zero_mask(RX1, RX2, NX, K), ZMY = zero_mask(RY1, RY2, NY, Q);
    static_assert(RX1 * RX2 == NX && RY1 * RY2 == NY, "radix split");
    static_assert(NX % RB == 0 && RB % 2 == 0 && NX % 2 == 0, "row batches");
    static_assert(SMEM_BYTES <= 232448, "plane does not fit in shared memory");
};

// Arrival on a counter with release semantics (everything this thread has observed, including the other threads'
// stores ordered before it by a CTA barrier, is visible to whoever acquires the new value).  Unlike
// __threadfence() + atomicAdd the thread does not wait for its stores to be acknowledged: it can exit at once.
__device__ __forceinline__ void arrive_release(unsigned* counter) {
    asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(counter) : "memory");
}

// Thread context of a phase function: the whole CTA.  (A two-units-per-CTA variant with one named barrier per
// group was measured in round 2: 67.5 against 57.3 us.)
struct CtaSync {
    __device__ __forceinline__ int tid() const { return (int)threadIdx.x; }
    __device__ __forceinline__ void sync() const { __syncthreads(); }
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
    unsigned* count;      // [s][m][z] arrival counters of the J node-units (monotonic: +J per call)
    const float2* twx;    // e^{+2 pi i t/NX}
    const float2* twy;
    float dkx, dky, scale;
    int Nz, Nl, Nm, Ns, J;
    // electromagnetic evaluations (gx_nonlinear_rhs_em) hand the chi kernels ready-made spectral planes
    // chi_{s,z,j}(k): phi then holds one plane per unit (s,z,j) and M one shared plane of ones
    int phi_by_unit, M_shared;
    int accumulate;       // inverse-Laguerre kernel: out += instead of out =
    unsigned a8_target;   // != 0 (row family): the node unit j = J-1 does a8 itself once count == a8_target - 1 (no third kernel)
    int ZG;               // row family: z values per block group of the unit order (divides Nz)
    // chained calls (row family, gx_api.cu nl_enqueue): `done` counts the bracket units, over all calls, that have
    // finished reading dchi; the chi grid of a call may overwrite its dchi buffer once done >= chi_need
    unsigned* done;
    unsigned chi_need;
    // Runge-Kutta stage folded into the separate inverse-Laguerre kernel (gx_ssprk3_step): st_out = a y0 + b (y + dt rhs)
    const float2* st_y0;
    const float2* st_y;
    float2* st_out;       // nullptr: off
    float st_a, st_b, st_dt;
    int cluster;          // row family: the J node units of an (s,m,z) are one thread-block cluster (a8 over distributed shared memory)
    unsigned* chi_ready;  // chained calls: [s][z][j] of the current dchi buffer, epoch of the call that wrote the plane
    unsigned chi_epoch;
};

// ------------------------------------------------------------------------------------------------
// inverse x transform of U(k) = (i kx - ky) f(k) on the 2*naky-1 non-zero columns.
// F: compact f, [NAKX][NAKY], in shared memory (STAGE) or global memory.
// Element classes of input n = n1*R2 + n2 are resolved at compile time per n1: always kept with
// kx >= 0, always kept with kx < 0, always padding, or decided by n2 at run time (at most two n1).
// For column q < 0 the reality condition gives f(a,q) = conj f(-a,-q): row index and the sign of the
// imaginary part flip, which keeps every address of the form base + compile-time offset.
struct NoMid { __device__ __forceinline__ void operator()() const {} };
// MID: called by every thread between the two passes (after the barrier): a place for work that only needs issue
// slots, e.g. cache prefetches of data the next phase will read.
template <class C, bool GLOBAL_F, class SY = CtaSync, class MID = NoMid>
__device__ __forceinline__ void x_inverse(float2* __restrict__ W, const float2* __restrict__ twx,
                                          float dkx, float dky, const float2* __restrict__ F, const SY sy = SY(),
                                          const MID mid = MID()) {
    constexpr int NX = C::NX, K = C::K, NCOL = C::NCOL, NAKY = C::NAKY, NAKX = C::NAKX;
    constexpr int R1 = C::RX1, R2 = C::RX2;
    // pass 1: for each (n2, column): DFT_R1 over n1 of input n = n1*R2+n2, twiddle, in-place slot
    for (int t = sy.tid(); t < R2 * NCOL; t += C::NT) {
        const int n2 = t / NCOL, c = t - n2 * NCOL;
        const bool neg = c >= NAKY;                       // column q < 0
        const int qa = neg ? NCOL - c : c;                // |q|
        const float kyq = neg ? -dky * (float)qa : dky * (float)qa;
        const float sgn = neg ? -1.f : 1.f;               // conj for q < 0
        // compact row of mode a (or of -a when q < 0), as base + n1 * step
        //   kx >= 0 branch, a = n:        q>=0: row  n            q<0: row NAKX - n   (n = 0 -> row 0)
        //   kx <  0 branch, a = n - NX:   q>=0: row  n - NX + NAKX  q<0: row NX - n
        const int stepP = neg ? -R2 * NAKY : R2 * NAKY;
        const float2* __restrict__ FP = F + (neg ? (NAKX - n2) * NAKY : n2 * NAKY) + qa;
        const float2* __restrict__ FN = F + (neg ? (NX - n2) * NAKY : (n2 - NX + NAKX) * NAKY) + qa;
        const float an2 = (float)n2, an2n = (float)(n2 - NX);   // integers: sums below are exact in fp32
        float2 v[R1];
#pragma unroll
        for (int n1 = 0; n1 < R1; ++n1) {
            const int lo = n1 * R2, hi = n1 * R2 + R2 - 1;           // range of n over n2 (compile time)
            const bool allP = hi <= K, someP = lo <= K;              // kept with kx >= 0
            const bool allN = lo >= NX - K, someN = hi >= NX - K;    // kept with kx < 0
            v[n1] = make_float2(0.f, 0.f);
            if (someP || someN) {
                float2 f = make_float2(0.f, 0.f);
                float kxa = 0.f;
                if (someP) {
                    const bool isP = allP || (lo + n2 <= K);
                    const float2* ptr = FP + n1 * stepP;
                    if (n1 == 0 && neg && n2 == 0) ptr = F + qa;     // mode a = 0: -a is row 0, not NAKX
                    if (isP) {
                        f = GLOBAL_F ? __ldg(ptr) : *ptr;
                        kxa = dkx * (an2 + (float)lo);
                    }
                }
                if (someN) {
                    const bool isN = allN || (lo + n2 >= NX - K);
                    if (isN) {
                        const float2* ptr = FN + n1 * stepP;
                        f = GLOBAL_F ? __ldg(ptr) : *ptr;
                        kxa = dkx * (an2n + (float)lo);
                    }
                }
                const float fy = sgn * f.y;
                v[n1] = make_float2(fmaf(-kyq, f.x, -kxa * fy), fmaf(kxa, f.x, -kyq * fy));
            }
        }
        dft<R1, +1, C::ZMX>(v);
#pragma unroll
        for (int k1 = 0; k1 < R1; ++k1)
            W[(k1 * R2 + n2) * NCOL + c] = k1 == 0 ? v[0] : cmul(v[k1], twx[n2 * k1]);
    }
    sy.sync();
    mid();
    // pass 2: for each (k1, column): DFT_R2 over n2; position k1*R2+k2 <- x = k1 + R1*k2
    for (int t = sy.tid(); t < R1 * NCOL; t += C::NT) {
        const int k1 = t / NCOL, c = t - k1 * NCOL;
        float2 v[R2];
#pragma unroll
        for (int n2 = 0; n2 < R2; ++n2) v[n2] = W[(k1 * R2 + n2) * NCOL + c];
        dft<R2, +1>(v);
#pragma unroll
        for (int k2 = 0; k2 < R2; ++k2) W[(k1 * R2 + k2) * NCOL + c] = v[k2];
    }
    sy.sync();
}

template <class C>
__device__ __forceinline__ void x_inverse_global_rw(float2* __restrict__ W, const float2* __restrict__ twx,
                                                    float dkx, float dky, const float2* F) {
    __threadfence_block();
    x_inverse<C, false>(W, twx, dkx, dky, F);        // plain ld: data was written by this CTA
}

// y inverse pass 1 for a batch of RB rows: W rows (2*naky-1 non-zero inputs) -> S[(k1*RY2+n2)*RB + r]
template <class C, bool PAIRED>
__device__ __forceinline__ void y_inverse_pass1(const float2* __restrict__ W, float2* __restrict__ S,
                                                const float2* __restrict__ twy, int bt) {
    constexpr int NX = C::NX, NY = C::NY, Q = C::Q, NCOL = C::NCOL, RB = C::RB, HB = C::HB;
    constexpr int R1 = C::RY1, R2 = C::RY2;
    for (int t = threadIdx.x; t < R2 * RB; t += C::NT) {
        const int n2 = t / RB, r = t - n2 * RB;
        const int row = !PAIRED ? bt * RB + r
                      : C::ADJ ? (r < HB ? bt * RB + 2 * r : bt * RB + 2 * (r - HB) + 1)
                               : (r < HB ? bt * HB + r : bt * HB + (r - HB) + NX / 2);
        const float2* __restrict__ Wr = W + row * NCOL;
        const float2* __restrict__ WP = Wr + n2;                  // ky >= 0: column n
        const float2* __restrict__ WN = Wr + n2 - NY + NCOL;      // ky <  0: column n - NY + NCOL
        float2 v[R1];
#pragma unroll
        for (int n1 = 0; n1 < R1; ++n1) {
            const int lo = n1 * R2, hi = n1 * R2 + R2 - 1;
            const bool allP = hi <= Q, someP = lo <= Q, allN = lo >= NY - Q, someN = hi >= NY - Q;
            v[n1] = make_float2(0.f, 0.f);
            if (someP && (allP || lo + n2 <= Q)) v[n1] = WP[lo];
            if (someN && (allN || lo + n2 >= NY - Q)) v[n1] = WN[lo];
        }
        dft<R1, +1, C::ZMY>(v);
#pragma unroll
        for (int k1 = 0; k1 < R1; ++k1)
            S[C::sidx(k1, n2, r)] = k1 == 0 ? v[0] : cmul(v[k1], twy[n2 * k1]);
    }
    __syncthreads();
}

// ---- transposed configurations (nl_row_kernels.cuh, RowCfg<..., TR = true>): the kernel works on the transposed
// plane (its x is the physical y and vice versa, so that the 64-point direction is the one held in registers), the
// arrays in memory keep the physical compact layout [ikx][ky], ikx in FFT order over 2Q+1 values, ky = 0..K.
// With f'(a, q) = f(kx = q, ky = a) and the reality condition f(-k) = conj f(k):
//   physical (kx >= 0, ky)      <-> internal (a = ky, q = kx)
//   physical (kx <  0, ky >  0) <-> conj of internal (a = -ky, q = -kx)
//   physical (kx =  0, ky >  0) also gives internal (a = -ky, q = 0) = conj;  physical (kx < 0, ky = 0) = conj internal (0, -kx).
template <class C>
__device__ __forceinline__ void tr_scatter(float2* __restrict__ S, const int i, const float2 v) {
    constexpr int NAKYP = C::K + 1;
    const int ikx = i / NAKYP, ky = i - ikx * NAKYP;
    const float2 vc = make_float2(v.x, -v.y);
    if (ikx <= C::Q) {
        S[ky * C::NAKY + ikx] = v;
        if (ikx == 0 && ky > 0) S[(C::NAKX - ky) * C::NAKY] = vc;
    } else if (ky > 0) {
        S[(C::NAKX - ky) * C::NAKY + (C::NCOL - ikx)] = vc;
    }
}
struct LinearStore {      // compact internal index = memory index
    __device__ __forceinline__ void operator()(float2* __restrict__ out, const int i, const int q, const int naky, const float2 v) const {
        out[i * naky + q] = v;
    }
};
template <class C> struct TrStore {      // internal (row i of the compact kx' order, q) -> physical [ikx][ky]
    __device__ __forceinline__ void operator()(float2* __restrict__ out, const int i, const int q, const int, const float2 v) const {
        constexpr int NAKYP = C::K + 1;
        const float2 vc = make_float2(v.x, -v.y);
        if (i <= C::K) {                                   // a = i >= 0: (kx = q, ky = i)
            out[q * NAKYP + i] = v;
            if (i == 0 && q > 0) out[(C::NCOL - q) * NAKYP] = vc;
        } else if (q > 0) {                                // a = i - NAKX < 0: (kx = -q, ky = NAKX - i)
            out[(C::NCOL - q) * NAKYP + (C::NAKX - i)] = vc;
        }
    }
};

// forward x transform on the naky kept columns; W holds Bhat(x, q) at permuted x positions.
// Writes the 2K+1 kept kx rows (compact order) times `scale` to out[i*NAKY + q].
template <class C, class SY = CtaSync, class ST = LinearStore>
__device__ __forceinline__ void x_forward(float2* __restrict__ W, const float2* __restrict__ twx,
                                          float2* __restrict__ out, float scale, const SY sy = SY(), const ST store = ST()) {
    constexpr int NX = C::NX, K = C::K, NCOL = C::NCOL, NAKY = C::NAKY, NAKX = C::NAKX;
    constexpr int R1 = C::RX1, R2 = C::RX2;
    for (int t = sy.tid(); t < R1 * NAKY; t += C::NT) {
        const int a = t / NAKY, q = t - a * NAKY;
        float2 v[R2];
#pragma unroll
        for (int b = 0; b < R2; ++b) v[b] = W[(a * R2 + b) * NCOL + q];
        dft<R2, -1>(v);
#pragma unroll
        for (int d = 0; d < R2; ++d)
            W[(a * R2 + d) * NCOL + q] = d == 0 ? v[0] : cmul_conj(v[d], twx[a * d]);
    }
    sy.sync();
    for (int t = sy.tid(); t < R2 * NAKY; t += C::NT) {
        // lanes run along q (contiguous in the compact layout); transposed configurations store along the row index
        // instead, which is n = d + R2*cc: there d is the fastest index of a warp
        const int d = C::TR ? t % R2 : t / NAKY, q = C::TR ? t / R2 : t - d * NAKY;
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
                if (i >= 0) store(out, i, q, NAKY, make_float2(v[cc].x * scale, v[cc].y * scale));
            }
        }
    }
}

// Programmatic dependent launch (sm_90+): the dependent grid may start while the primary still runs;
// it must not touch the primary's output before pdl_wait().  Both are no-ops without the launch attribute.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;"); }

// S[i] = sum_l coef[l] * planes[l*lstride + i], i < NK: U positions x 2 planes of independent 8-byte
// loads in flight per thread (the loop is latency-bound otherwise: ncu r01 showed 35% of the bracket
// kernel's stall samples here).
template <class C>
__device__ __forceinline__ void stage_combine(float2* __restrict__ S, const float2* __restrict__ planes,
                                              size_t lstride, const float* __restrict__ coef, int Nl) {
    // U positions x LB planes per round trip, U chosen so that the positions of a thread take the fewest rounds of at
    // most 12 (stellarator plane: 22 positions per thread = 2 rounds of 11, 22 loads in flight; measured against
    // 4 x 4: 3 982 -> 3 865 us per call, 6 x 4: 3 930, 6 x 8: 3 886, 3 x 11: 3 881)
    constexpr int NK = C::NK, NT = C::NT, LB = 2;
    constexpr int PER = (NK + NT - 1) / NT, ROUNDS = (PER + 11) / 12, U = (PER + ROUNDS - 1) / ROUNDS;
    for (int i0 = threadIdx.x; i0 < NK; i0 += U * NT) {
        float2 acc[U];
#pragma unroll
        for (int u = 0; u < U; ++u) acc[u] = make_float2(0.f, 0.f);
        for (int l0 = 0; l0 < Nl; l0 += LB) {
            float2 f[LB][U];
#pragma unroll
            for (int dl = 0; dl < LB; ++dl)
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    const int i = i0 + u * NT;
                    f[dl][u] = (l0 + dl < Nl && i < NK) ? __ldg(planes + (size_t)(l0 + dl) * lstride + i)
                                                        : make_float2(0.f, 0.f);
                }
#pragma unroll
            for (int dl = 0; dl < LB; ++dl) {
                const float t = (l0 + dl < Nl) ? __ldg(coef + l0 + dl) : 0.f;
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    acc[u].x = fmaf(t, f[dl][u].x, acc[u].x);
                    acc[u].y = fmaf(t, f[dl][u].y, acc[u].y);
                }
            }
        }
#pragma unroll
        for (int u = 0; u < U; ++u)
            if (i0 + u * NT < NK) S[i0 + u * NT] = acc[u];
    }
}

// ---- TMA bulk staging (cp.async.bulk + mbarrier): the Nl compact planes of one (s,m,z) are contiguous
// 16-byte aligned chunks of NK*8 bytes; one elected thread copies them into the (still unused) W+S region,
// everyone waits on the mbarrier, combines them with the Laguerre row T[j][.] in registers and, after a
// barrier, writes gt into S.  No per-element global load instruction or address arithmetic is issued.
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, unsigned long long* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

template <class C, class SY = CtaSync>
__device__ __forceinline__ void stage_combine_tma(float2* __restrict__ raw, float2* __restrict__ S,
                                                  unsigned long long* bar, unsigned& parity,
                                                  const float2* __restrict__ planes,
                                                  size_t lstride, const float* __restrict__ coef, int Nl,
                                                  const SY sy = SY()) {
    constexpr int NK = C::NKP, NT = C::NT, NK2 = NK / 2;     // planes as they lie in memory
    constexpr int CAP = (C::W_ELEMS + C::S_ELEMS) / NK;          // planes per chunk
    constexpr int PER = (NK2 + NT - 1) / NT;                     // float4 (2 complex) per thread
    const int tid = sy.tid();
    static_assert(CAP >= 1 && NK % 2 == 0, "TMA staging needs 16-byte planes that fit");
    const float4* __restrict__ raw4 = reinterpret_cast<const float4*>(raw) + tid;
    float4 acc[PER];
#pragma unroll
    for (int u = 0; u < PER; ++u) acc[u] = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int l0 = 0; l0 < Nl; l0 += CAP) {
        const int nl = min(CAP, Nl - l0);
        if (tid == 0) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            mbar_expect_tx(bar, (unsigned)(nl * NK * sizeof(float2)));
            for (int l = 0; l < nl; ++l)
                bulk_g2s(raw + l * NK, planes + (size_t)(l0 + l) * lstride, NK * sizeof(float2), bar);
        }
        mbar_wait(bar, parity);
        parity ^= 1u;
        for (int l = 0; l < nl; ++l) {
            const float t = coef[l0 + l];
            const float4* __restrict__ src = raw4 + l * NK2;
#pragma unroll
            for (int u = 0; u < PER; ++u) {
                if ((u + 1) * NT <= NK2 || tid + u * NT < NK2) {
                    const float4 f = src[u * NT];
                    acc[u].x = fmaf(t, f.x, acc[u].x);
                    acc[u].y = fmaf(t, f.y, acc[u].y);
                    acc[u].z = fmaf(t, f.z, acc[u].z);
                    acc[u].w = fmaf(t, f.w, acc[u].w);
                }
            }
        }
        sy.sync();                                             // raw region consumed
    }
    if constexpr (C::TR) {
#pragma unroll
        for (int u = 0; u < PER; ++u)
            if ((u + 1) * NT <= NK2 || tid + u * NT < NK2) {
                const int i = 2 * (tid + u * NT);
                tr_scatter<C>(S, i, make_float2(acc[u].x, acc[u].y));
                tr_scatter<C>(S, i + 1, make_float2(acc[u].z, acc[u].w));
            }
    } else {
        float4* __restrict__ S4 = reinterpret_cast<float4*>(S) + tid;
#pragma unroll
        for (int u = 0; u < PER; ++u)
            if ((u + 1) * NT <= NK2 || tid + u * NT < NK2) S4[u * NT] = acc[u];
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
    const float2* __restrict__ phi = p.phi + (size_t)(p.phi_by_unit ? unit : z) * C::NK;
    const float* __restrict__ M = p.M + (size_t)(p.M_shared ? 0 : unit) * C::NK;
    pdl_launch_dependents();        // the bracket kernel's prologue (a2-a4 x part) does not read dchi
    load_twiddles<C>(twx, twy, p);
    if constexpr (C::STAGE) {
        constexpr int U = 4;
        for (int i0 = threadIdx.x; i0 < C::NK; i0 += U * C::NT) {
            float2 f[U];
            float m[U];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int i = i0 + u * C::NT;
                f[u] = i < C::NK ? __ldg(phi + i) : make_float2(0.f, 0.f);
                m[u] = i < C::NK ? __ldg(M + i) : 0.f;
            }
#pragma unroll
            for (int u = 0; u < U; ++u)
                if (i0 + u * C::NT < C::NK) S[i0 + u * C::NT] = make_float2(f[u].x * m[u], f[u].y * m[u]);
        }
        __syncthreads();
        x_inverse<C, false>(W, twx, p.dkx, p.dky, S);
    } else {
        // plane too large to stage: chi = M.Phi goes through this unit's own (not yet written) dchi slot
        float2* __restrict__ tmp = p.dchi + (size_t)unit * C::NX * C::NY;
        for (int i = threadIdx.x; i < C::NK; i += C::NT) {
            const float2 f = __ldg(phi + i);
            const float m = __ldg(M + i);
            tmp[i] = make_float2(f.x * m, f.y * m);
        }
        __syncthreads();
        x_inverse_global_rw<C>(W, twx, p.dkx, p.dky, tmp);
    }
    float2* __restrict__ dchi = p.dchi + (size_t)unit * C::NX * C::NY;
    constexpr int R1 = C::RY1, R2 = C::RY2, RB = C::RB;
    for (int bt = 0; bt < C::NBATCH; ++bt) {
        y_inverse_pass1<C, false>(W, S, twy, bt);
        for (int t = threadIdx.x; t < R1 * RB; t += C::NT) {
            const int k1 = t / RB, r = t - k1 * RB;
            float2 v[R2];
#pragma unroll
            for (int n2 = 0; n2 < R2; ++n2) v[n2] = S[C::sidx(k1, n2, r)];
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

    __shared__ unsigned long long stage_bar;
    __shared__ float Tsh[16];
    unsigned bar_parity = 0;
    if constexpr (C::STAGE && C::NK % 2 == 0) {
        if (threadIdx.x == 0) mbar_init(&stage_bar, 1);
        if (threadIdx.x < p.Nl) Tsh[threadIdx.x] = __ldg(Tj + threadIdx.x);
        __syncthreads();
    }
    pdl_launch_dependents();        // inverse-Laguerre grid may become resident once our last wave runs
    load_twiddles<C>(twx, twy, p);
    // ---- a2: forward Laguerre transform l -> node j, fused into the load
    if constexpr (C::STAGE) {
        if constexpr (C::NK % 2 == 0) stage_combine_tma<C>(W, S, &stage_bar, bar_parity, g0, lstride, Tsh, p.Nl);
        else stage_combine<C>(S, g0, lstride, Tj, p.Nl);
        __syncthreads();
        x_inverse<C, false>(W, twx, p.dkx, p.dky, S);
    } else {
        // plane too large to stage in shared memory: gt goes through this unit's own bhat slot
        // (written by this CTA, read back by this CTA after the barrier; overwritten by the result later)
        float2* __restrict__ tmp = p.bhat + (size_t)unit * NK;
        stage_combine<C>(tmp, g0, lstride, Tj, p.Nl);
        __syncthreads();
        x_inverse_global_rw<C>(W, twx, p.dkx, p.dky, tmp);
    }

    const float2* dchi = p.dchi + (size_t)szj * NX * NY;   // written by the overlapping chi grid: no __restrict__/ld.nc
    pdl_wait();                     // chi planes of this call are complete and visible from here on
    for (int bt = 0; bt < C::NBATCH; ++bt) {
        // ---- a4 (y part): rows p and p+NX/2 of the batch
        y_inverse_pass1<C, true>(W, S, twy, bt);
        if constexpr (2 * R1 * HB <= C::NT) {
            // Small batches (the plane fills shared memory): R1*HB items would keep a quarter of the CTA busy through three
            // transforms.  One thread per ROW does the last inverse pass and the bracket and leaves the real result in
            // the slots it has just read; after a barrier one thread per row PAIR does the first forward pass.
            for (int t = threadIdx.x; t < R1 * RB; t += C::NT) {
                const int k1 = t / RB, r = t - k1 * RB;
                const int h = r / HB, rp = r - h * HB;
                const int row = C::ADJ ? bt * RB + 2 * rp + h : bt * HB + rp + h * (NX / 2);
                float2 v[R2];
                float2 dv[R2];                                       // requested before the transform (L2 round trip under it)
#pragma unroll
                for (int k2 = 0; k2 < R2; ++k2) dv[k2] = __ldcg(dchi + (size_t)(k1 * R2 + k2) * NX + row);
#pragma unroll
                for (int n2 = 0; n2 < R2; ++n2) v[n2] = S[C::sidx(k1, n2, r)];
                dft<R2, +1>(v);
#pragma unroll
                for (int k2 = 0; k2 < R2; ++k2) {
                    const float2 d = dv[k2];
                    S[C::sidx(k1, k2, r)] = make_float2(fmaf(d.y, v[k2].x, -d.x * v[k2].y), 0.f);
                }
            }
            __syncthreads();
            for (int t = threadIdx.x; t < R1 * HB; t += C::NT) {
                const int k1 = t / HB, rp = t - k1 * HB;
                float2 c[R2];
#pragma unroll
                for (int k2 = 0; k2 < R2; ++k2)
                    c[k2] = make_float2(S[C::sidx(k1, k2, rp)].x, S[C::sidx(k1, k2, rp + HB)].x);
                dft<R2, -1>(c);
#pragma unroll
                for (int d = 0; d < R2; ++d)
                    S[C::sidx(k1, d, rp)] = d == 0 ? c[0] : cmul_conj(c[d], twy[k1 * d]);
            }
        } else {
            // ---- a4 (last pass) + a5 bracket + a6 (first forward pass), all in registers
            for (int t = threadIdx.x; t < R1 * HB; t += C::NT) {
                const int k1 = t / HB, rp = t - k1 * HB;
                float2 c[R2];
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const int r = rp + h * HB;
                    const int row = C::ADJ ? bt * RB + 2 * rp + h : bt * HB + rp + h * (NX / 2);
                    float2 v[R2];
                    float2 dv[R2];                                   // requested before the transform: the L2 round trip passes under it
#pragma unroll
                    for (int k2 = 0; k2 < R2; ++k2) dv[k2] = __ldcg(dchi + (size_t)(k1 * R2 + k2) * NX + row);
#pragma unroll
                    for (int n2 = 0; n2 < R2; ++n2) v[n2] = S[C::sidx(k1, n2, r)];
                    dft<R2, +1>(v);
#pragma unroll
                    for (int k2 = 0; k2 < R2; ++k2) {
                        const float2 d = dv[k2];
                        const float b = fmaf(d.y, v[k2].x, -d.x * v[k2].y);   // d_y chi d_x g - d_x chi d_y g
                        if (h == 0) c[k2].x = b; else c[k2].y = b;
                    }
                }
                dft<R2, -1>(c);
#pragma unroll
                for (int d = 0; d < R2; ++d)
                    S[C::sidx(k1, d, rp)] = d == 0 ? c[0] : cmul_conj(c[d], twy[k1 * d]);
            }
        }
        __syncthreads();
        if constexpr (2 * R1 * HB <= C::NT) {
            // small batches: one thread per (class d, row pair) does the last forward pass in place, then, after a
            // barrier, one thread per kept (ky, row pair) separates the packed rows (the fused loop below would keep
            // (R2/2+1)*HB threads -- three warps of twelve -- busy through two transforms; it took a third of the kernel)
            for (int t = threadIdx.x; t < R2 * HB; t += C::NT) {
                const int d = t / HB, rp = t - d * HB;
                float2 u[R1];
#pragma unroll
                for (int a = 0; a < R1; ++a) u[a] = S[C::sidx(a, d, rp)];
                dft<R1, -1>(u);
#pragma unroll
                for (int a = 0; a < R1; ++a) S[C::sidx(a, d, rp)] = u[a];
            }
            __syncthreads();
            for (int t = threadIdx.x; t < (Q + 1) * HB; t += C::NT) {
                const int k = t / HB, rp = t - k * HB;
                const int d = k % R2, cc = k / R2;
                const int dp = (R2 - d) % R2, cp = d == 0 ? (R1 - cc) % R1 : R1 - 1 - cc;     // NY - k = dp + R2*cp
                const float2 A = S[C::sidx(cc, d, rp)], B = S[C::sidx(cp, dp, rp)];
                float2* __restrict__ W0 = W + (C::ADJ ? bt * RB + 2 * rp : bt * HB + rp) * NCOL;
                float2* __restrict__ W1 = W0 + (C::ADJ ? 1 : NX / 2) * NCOL;
                W0[k] = make_float2(0.5f * (A.x + B.x), 0.5f * (A.y - B.y));
                W1[k] = make_float2(0.5f * (A.y + B.y), 0.5f * (B.x - A.x));
            }
        } else {
            // ---- a6 (last y pass) + a7 (keep ky <= Q) + separation of the packed row pair
            for (int t = threadIdx.x; t < (R2 / 2 + 1) * HB; t += C::NT) {
                const int dd = t / HB, rp = t - dd * HB;
                const int d0 = dd, d1 = (R2 - dd) % R2;
                float2 u0[R1], u1[R1];
#pragma unroll
                for (int a = 0; a < R1; ++a) u0[a] = S[C::sidx(a, d0, rp)];
                dft<R1, -1>(u0);
                if (d1 != d0) {
#pragma unroll
                    for (int a = 0; a < R1; ++a) u1[a] = S[C::sidx(a, d1, rp)];
                    dft<R1, -1>(u1);
                } else {
#pragma unroll
                    for (int a = 0; a < R1; ++a) u1[a] = u0[a];
                }
                float2* __restrict__ W0 = W + (C::ADJ ? bt * RB + 2 * rp : bt * HB + rp) * NCOL;
                float2* __restrict__ W1 = W0 + (C::ADJ ? 1 : NX / 2) * NCOL;
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
        }
        __syncthreads();
    }
    // ---- a6 (x part) + a7 (keep |kx| <= K)
    x_forward<C>(W, twx, p.bhat + (size_t)unit * NK, p.scale);

    // ---- publish: this node's Bhat plane is complete (release: stores -> barrier -> fence -> atomic).
    // The inverse-Laguerre grid, already resident under PDL, waits per (s,m,z) on this counter.
    __syncthreads();                 // orders every thread's stores before thread 0's gpu-scope fence (cumulative)
    if (threadIdx.x == 0) arrive_release(p.count + (s * p.Nm + m) * p.Nz + z);
}

// ================================================================================================
// a8: out[s,m,l,z,k] = - sum_j Tinv[l][j] Bhat[s,z,j,m,k].  VEC = 2 complex per thread (16-byte accesses)
// when nk is even, else 1.  Launched with PDL: blocks become resident during the bracket kernel's last
// wave and wait until the J node-units of their (s,m,z) have arrived (count >= target; the counters
// grow by J per call, target = J * call number, so nothing is ever reset).
// MODE 0: out = -N; 1: out += -N (gx_rhs: linear terms already there); 2: Runge-Kutta stage on top of mode 1.
template <int MAXL, int MAXJ, int VEC, int MODE = 0>
__global__ void __launch_bounds__(256) laguerre_inverse_kernel(const NlParams p, int nk, unsigned target) {
    using V = typename std::conditional<VEC == 2, float4, float2>::type;
    const int kv = blockIdx.x * blockDim.x + threadIdx.x;      // index in units of VEC complex
    // blocks are handed out in the order in which the bracket grid completes the (s,m,z): z before m (a block that
    // waits for a late z would otherwise hold one of the few slots left beside the bracket CTAs)
    const int m = blockIdx.y % p.Nm;
    const int z = (blockIdx.y / p.Nm) % p.Nz;
    const int s = blockIdx.y / (p.Nz * p.Nm);
    const int smz = (s * p.Nm + m) * p.Nz + z;
    __shared__ float Ti[MAXL * MAXJ];
    for (int i = threadIdx.x; i < p.Nl * p.J; i += blockDim.x) Ti[i] = -__ldg(p.Tinv + i);   // out = -N
    if (threadIdx.x == 0) {
        const volatile unsigned* c = p.count + smz;
        while ((int)(*c - target) < 0) __nanosleep(200);
        __threadfence();
    }
    __syncthreads();
    const int nkv = nk / VEC;
    if (kv >= nkv) return;
    V b[MAXJ];
#pragma unroll
    for (int j = 0; j < MAXJ; ++j)
        if (j < p.J)
            b[j] = __ldcg(reinterpret_cast<const V*>(p.bhat + ((size_t)((s * p.Nz + z) * p.J + j) * p.Nm + m) * nk) + kv);
    // Moments in groups of four: what the result is combined with (the linear terms already in out: gx_rhs; the two
    // states of a Runge-Kutta stage: gx_ssprk3_step) is requested for the whole group before its first store.
    constexpr bool stage = MODE == 2, accumulate = MODE >= 1;
#pragma unroll
    for (int l0 = 0; l0 < MAXL; l0 += 4) {
        V prev[accumulate ? 4 : 1], vy0[stage ? 4 : 1], vy[stage ? 4 : 1];
#pragma unroll
        for (int dl = 0; dl < 4; ++dl) {
            const int l = l0 + dl;
            if (l < p.Nl && accumulate) {
                const size_t idx = (((size_t)(s * p.Nm + m) * p.Nl + l) * p.Nz + z) * nk;
                prev[dl] = *(reinterpret_cast<const V*>(p.out + idx) + kv);
                if constexpr (stage) {
                    vy0[dl] = *(reinterpret_cast<const V*>(p.st_y0 + idx) + kv);
                    vy[dl] = *(reinterpret_cast<const V*>(p.st_y + idx) + kv);
                }
            }
        }
#pragma unroll
        for (int dl = 0; dl < 4; ++dl) {
            const int l = l0 + dl;
            if (l < p.Nl) {
                float acc[2 * VEC];
#pragma unroll
                for (int c = 0; c < 2 * VEC; ++c) acc[c] = 0.f;
#pragma unroll
                for (int j = 0; j < MAXJ; ++j)
                    if (j < p.J) {
                        const float t = Ti[l * p.J + j];
                        const float* bj = reinterpret_cast<const float*>(&b[j]);
#pragma unroll
                        for (int c = 0; c < 2 * VEC; ++c) acc[c] = fmaf(t, bj[c], acc[c]);
                    }
                const size_t idx = (((size_t)(s * p.Nm + m) * p.Nl + l) * p.Nz + z) * nk;
                if constexpr (accumulate) {          // gx_rhs: the linear terms are already in out (written concurrently)
                    const float* pv = reinterpret_cast<const float*>(&prev[dl]);
#pragma unroll
                    for (int c = 0; c < 2 * VEC; ++c) acc[c] += pv[c];
                }
                if constexpr (stage) {               // SSP-RK3 stage: st_out = a y0 + b (y + dt rhs); rhs itself is not stored
                    const float* a0 = reinterpret_cast<const float*>(&vy0[dl]);
                    const float* a1 = reinterpret_cast<const float*>(&vy[dl]);
#pragma unroll
                    for (int c = 0; c < 2 * VEC; ++c) acc[c] = fmaf(p.st_a, a0[c], p.st_b * fmaf(p.st_dt, acc[c], a1[c]));
                    *(reinterpret_cast<V*>(p.st_out + idx) + kv) = *reinterpret_cast<V*>(acc);
                } else {
                    *(reinterpret_cast<V*>(p.out + idx) + kv) = *reinterpret_cast<V*>(acc);
                }
            }
        }
    }
}

}  // namespace gx
