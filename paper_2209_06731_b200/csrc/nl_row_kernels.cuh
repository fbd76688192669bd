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

// Development builds (-DGX_PHASE_TIMING): %globaltimer at the phase boundaries of EVERY bracket CTA (slot 7: SM id),
// read back with gx_debug_cta_log(): the timeline of a whole launch (waves, tail, closers).
#ifdef GX_PHASE_TIMING
static __device__ long long gx_cta_log[4 * 8192 * 16];     // [call & 3][block][slot]
static __device__ long long gx_chi_log[4 * 256 * 4];        // [call & 3][block][start, before the done wait, after it, end]
__device__ __forceinline__ long long gx_globaltimer() { long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t; }
__device__ __forceinline__ long long gx_smid() { unsigned s; asm volatile("mov.u32 %0, %%smid;" : "=r"(s)); return (long long)s; }
#define GX_CTA(i) do { if (threadIdx.x == 0 && blockIdx.x < 8192) gx_cta_log[(((p.a8_target / (unsigned)p.J) & 3u) * 8192 + blockIdx.x) * 16 + (i)] = (i) == 7 ? gx_smid() : gx_globaltimer(); } while (0)
#define GX_CHI(i) do { if (threadIdx.x == 0 && blockIdx.x < 256) gx_chi_log[(((p.a8_target / (unsigned)p.J) & 3u) * 256 + blockIdx.x) * 4 + (i)] = gx_globaltimer(); } while (0)
#else
#define GX_CTA(i) do { } while (0)
#define GX_CHI(i) do { } while (0)
#endif

// TR_ = true: the kernel's (NX, NY) is the TRANSPOSE of the physical plane (physical Nx = NY = 64, Ny = NX): the
// 64-point direction is always the one held in registers.  Memory keeps the physical compact layout (NKP elements
// per plane); the transposition happens where a plane enters (tr_scatter) and leaves (TrStore) shared memory, the
// host swaps dkx / dky and flips the sign of the bracket (nl_kernels.cuh, gx_api.cu).
template <int NX_, int NY_, int RX1_, int RX2_, int NT_, int MINB_, bool TR_ = false>
struct RowCfg {
    static constexpr int NX = NX_, NY = NY_, RX1 = RX1_, RX2 = RX2_, NT = NT_, MINB = MINB_;
    static constexpr bool TR = TR_;
    static constexpr int K = (NX - 1) / 3, Q = (NY - 1) / 3;
    static constexpr int NAKX = 2 * K + 1, NAKY = Q + 1, NCOL = 2 * Q + 1, NK = NAKX * NAKY;
    static constexpr int NKP = TR ? NCOL * (K + 1) : NK;         // plane in memory: [2Q+1 kx][K+1 ky] when transposed
    static constexpr int NKM = NK > NKP ? NK : NKP;
    static constexpr int W_ELEMS = NX * NCOL;
    // compact plane after the Laguerre combine; padded so that W + S hold 4 raw planes for the TMA staging
    static constexpr int S_MIN = 4 * NKM > W_ELEMS ? 4 * NKM - W_ELEMS : 0;
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
    static_assert(RX1 * RX2 == NX && NK % 2 == 0 && NKP % 2 == 0, "radix split / 16-byte planes");
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

// 64-point forward transform of the real sequence b -> TWICE the Q+1 kept coefficients into Wr[0..Q] (the factor
// 1/2 of the even/odd separation is folded into NlParams::scale by the host: 6 instructions fewer per coefficient).
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
        // 2E = Z[k] + conj Z[32-k] (even samples), 2O = (Z[k] - conj Z[32-k])/i (odd samples), X[k] = E + w^k O
        const float2 e = make_float2(a.x + c.x, a.y - c.y);
        const float2 o = make_float2(a.y + c.y, c.x - a.x);
        if (k == 0) {
            Wr[0] = cadd(e, o);
        } else {
            const float wr = (float)cos192(3 * k), wi = -(float)sin192(3 * k);     // w = e^{-2 pi i k/64}
            Wr[k] = make_float2(fmaf(-o.y, wi, fmaf(o.x, wr, e.x)), fmaf(o.y, wr, fmaf(o.x, wi, e.y)));
        }
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
    const float2* __restrict__ phi = p.phi + (size_t)(p.phi_by_unit ? unit : z) * C::NKP;
    const float* __restrict__ M = p.M + (size_t)(p.M_shared ? 0 : unit) * C::NKP;
    pdl_launch_dependents();
    GX_CHI(0);
    for (int i = threadIdx.x; i < C::NX; i += C::NT) twx[i] = p.twx[i];
    for (int i = threadIdx.x; i < C::NKP; i += C::NT) {
        const float2 f = __ldg(phi + i);
        const float m = __ldg(M + i);
        if constexpr (C::TR) tr_scatter<C>(S, i, make_float2(f.x * m, f.y * m));
        else S[i] = make_float2(f.x * m, f.y * m);
    }
    __syncthreads();
    x_inverse<C, false>(W, twx, p.dkx, p.dky, S);
    GX_CHI(1);
    if (p.done) {
        // Launched with the PDL attribute, this grid starts under the tail of the previous call's bracket grid.  It
        // writes the dchi buffer that the call BEFORE the previous one read: wait until all of that call's units
        // have left their row phase (normally long ago; x_inverse above ends with a CTA barrier, the one below
        // publishes thread 0's observation).
        if (threadIdx.x == 0) {
            unsigned c;
            do {
                asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(c) : "l"(p.done) : "memory");
                if ((int)(c - p.chi_need) < 0) __nanosleep(200);
            } while ((int)(c - p.chi_need) < 0);
        }
        __syncthreads();
    }
    GX_CHI(2);
    float2* __restrict__ dchi = p.dchi + (size_t)unit * C::NX * C::NY;
    for (int row = threadIdx.x; row < C::NX; row += C::NT) {
        float2 v[64];
        row_inverse<C>(W + row * C::NCOL, v);
#pragma unroll
        for (int y = 0; y < 64; ++y) dchi[y * C::NX + row] = v[y];
    }
    // Unchained launches keep the transitive order "bracket N+1 past its pdl_wait => chi N+1 complete => call N
    // complete"; chained ones (p.done) order the reuse of dchi, bhat and out through counters instead, so that the
    // next call's units can run under this call's tail.
    if (!p.done) pdl_wait();
    else {
        // chained: publish this plane (release: stores -> barrier -> release store of the flag); its bracket units wait for the
        // flag, not for the whole grid
        __syncthreads();
        if (threadIdx.x == 0)
            asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p.chi_ready + unit), "r"(p.chi_epoch) : "memory");
    }
    GX_CHI(3);
}

// a8 by the LAST node unit (j = J-1) of an (s,m,z), after its own plane is in bhat like everyone else's:
// out_l = - sum_j Tinv[l][j] Bhat_j.  The J-1 other node units were dispatched earlier (lower block indices); thread 0
// waits for their arrivals and fetches min(J, CAP) node planes with bulk copies into the (now free) W + S region, a
// last plane comes through registers.  Deliberately small, rolled code: it runs in one CTA out of J, so its
// instructions are cold in the instruction cache (a fully unrolled fused variant spent 7 us per closer on fetches).
// J <= CAP + 1 and Nl <= 4 (the host falls back to the separate inverse-Laguerre kernel otherwise).
template <class C, class SY>
__device__ __noinline__ void closer_sum(float2* __restrict__ raw, const float2* bh, const size_t jstride, float2* __restrict__ out0,
                                        const size_t lstride, const float* __restrict__ Tinv, const int J, const int Nl,
                                        const unsigned* cnt, const unsigned want, unsigned long long* bar, const unsigned parity,
                                        const SY sy, const NlParams& p) {
    constexpr int NK = C::NKP, NK2 = NK / 2, NT = C::NT;      // node planes lie in memory in the physical layout
    constexpr int CAP = (C::W_ELEMS + C::S_ELEMS) / NK;
    __shared__ float Tsm[4 * 8];              // -Tinv[l][j] (out = -N), zero-padded to [4][8]
    const int tid = sy.tid();
    if (tid < 32) {
        const int l = tid >> 3, jn = tid & 7;
        Tsm[tid] = (l < Nl && jn < J) ? -__ldg(Tinv + l * J + jn) : 0.f;
    }
    const int nt = min(J, CAP);
    // plane CAP (this unit's own plane when J = CAP + 1) through registers, requested first: the round trip to L2
    // (about 1 us under this kernel's load) passes while thread 0 waits and the bulk copies arrive
    constexpr int PER = (NK2 + NT - 1) / NT;
    float4 e[PER];
    {
        const float4* last4 = reinterpret_cast<const float4*>(bh + (size_t)CAP * jstride) + tid;
#pragma unroll
        for (int u = 0; u < PER; ++u)
            e[u] = (J > CAP && tid + u * NT < NK2) ? __ldcg(last4 + u * NT) : make_float4(0.f, 0.f, 0.f, 0.f);
    }
    GX_CTA(8);
    if (tid == 0) {
        unsigned c;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(c) : "l"(cnt) : "memory");
            if (c != want) __nanosleep(64);
        } while (c != want);
        GX_CTA(9);
        // the bulk copies (async proxy) read what other CTAs stored through the generic proxy; W + S were last
        // touched through the generic proxy by this CTA (x_forward, ordered by the barrier before this call)
        if (J <= CAP) __threadfence();        // this unit's own plane is among the copied ones
        asm volatile("fence.proxy.async;" ::: "memory");
        mbar_expect_tx(bar, (unsigned)(nt * NK * sizeof(float2)));
        for (int jn = 0; jn < nt; ++jn) bulk_g2s(raw + jn * NK, bh + jn * jstride, NK * sizeof(float2), bar);
    }
    sy.sync();                                // thread 0's acquire reaches everyone; Tsm complete
    GX_CTA(10);
    mbar_wait(bar, parity);
    GX_CTA(11);
    const float4* __restrict__ raw4 = reinterpret_cast<const float4*>(raw) + tid;
    float4* out4 = reinterpret_cast<float4*>(out0) + tid;
    const size_t lstride4 = lstride / 2;
#pragma unroll
    for (int u = 0; u < PER; ++u) {
        if (tid + u * NT < NK2) {
            float4 acc[4];
#pragma unroll
            for (int l = 0; l < 4; ++l) {
                const float t = Tsm[l * 8 + CAP];
                acc[l] = make_float4(t * e[u].x, t * e[u].y, t * e[u].z, t * e[u].w);
            }
#pragma unroll
            for (int jn = 0; jn < CAP; ++jn) {
                if (jn < nt) {
                    const float4 b = raw4[jn * NK2 + u * NT];
#pragma unroll
                    for (int l = 0; l < 4; ++l) {
                        const float t = Tsm[l * 8 + jn];
                        acc[l].x = fmaf(t, b.x, acc[l].x);
                        acc[l].y = fmaf(t, b.y, acc[l].y);
                        acc[l].z = fmaf(t, b.z, acc[l].z);
                        acc[l].w = fmaf(t, b.w, acc[l].w);
                    }
                }
            }
#pragma unroll
            for (int l = 0; l < 4; ++l)
                if (l < Nl) out4[l * lstride4 + u * NT] = acc[l];
        }
    }
    GX_CTA(12);
}

// ---- thread-block clusters (MODE 2 of bracket_row_kernel): the J node units of one (s,m,z) form one cluster, keep
// their Bhat_j planes in shared memory and do a8 over distributed shared memory -- no bhat workspace, no closer.
__device__ __forceinline__ unsigned cluster_ctarank() { unsigned r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ float4 ld_dsmem_f4(const void* local_smem_ptr, const unsigned rank) {
    unsigned ra;
    float4 v;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(ra) : "r"(smem_u32(local_smem_ptr)), "r"(rank));
    asm volatile("ld.shared::cluster.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(ra) : "memory");
    return v;
}
__device__ __forceinline__ void arrive_release_n(unsigned* counter, const unsigned n) {
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(counter), "r"(n) : "memory");
}

// a8 of one (s,m,z) by its cluster: CTA `rank` owns every J-th group of NT float4 slots of the plane, reads that
// group from the S region of all J CTAs and writes out_l = - sum_j Tinv[l][j] Bhat_j.  J <= 8, Nl <= 4.
template <class C, class SY>
__device__ __noinline__ void cluster_laguerre_inverse(const float2* S, float2* __restrict__ out0, const size_t lstride,
                                                      const float* __restrict__ Tinv, const int J, const int Nl,
                                                      const unsigned rank, const SY sy) {
    constexpr int NK2 = C::NKP / 2, NT = C::NT;
    __shared__ float Tsm[4 * 8];              // -Tinv[l][j] (out = -N), zero-padded to [4][8]
    const int tid = sy.tid();
    if (tid < 32) {
        const int l = tid >> 3, jn = tid & 7;
        Tsm[tid] = (l < Nl && jn < J) ? -__ldg(Tinv + l * J + jn) : 0.f;
    }
    sy.sync();
    const float4* S4 = reinterpret_cast<const float4*>(S);
    float4* out4 = reinterpret_cast<float4*>(out0);
    const size_t lstride4 = lstride / 2;
    for (int i = (int)rank * NT + tid; i < NK2; i += J * NT) {
        float4 b[8];
#pragma unroll
        for (int jn = 0; jn < 8; ++jn)
            b[jn] = jn < J ? ld_dsmem_f4(S4 + i, (unsigned)jn) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
        for (int l = 0; l < 4; ++l) {
            if (l < Nl) {
                float4 a = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
                for (int jn = 0; jn < 8; ++jn) {
                    const float t = Tsm[l * 8 + jn];
                    a.x = fmaf(t, b[jn].x, a.x);
                    a.y = fmaf(t, b[jn].y, a.y);
                    a.z = fmaf(t, b[jn].z, a.z);
                    a.w = fmaf(t, b[jn].w, a.w);
                }
                out4[l * lstride4 + i] = a;
            }
        }
    }
}

// unit = (((s*(Nz/ZG) + zg)*J + j)*ZG + zi)*Nm + m, z = zg*ZG + zi: the Nm units that share a chi plane stay
// neighbours, the J node units of one (s,m,z) lie ZG*Nm blocks apart (the last one, which does a8 in fused calls,
// starts late enough to find most of the other planes complete)
// Cluster mode: unit = ((s*Nz + z)*Nm + m)*J + j: the J node units of an (s,m,z) are the CTAs of one cluster.
struct UnitIdx { int s, m, z, j, szj; };
template <int MODE>
__device__ __forceinline__ UnitIdx decode_unit(const NlParams& p, const int unit) {
    UnitIdx ix;
    if (MODE == 2) {
        ix.j = unit % p.J;
        int r = unit / p.J;
        ix.m = r % p.Nm; r /= p.Nm;
        ix.z = r % p.Nz;
        ix.s = r / p.Nz;
        ix.szj = (ix.s * p.Nz + ix.z) * p.J + ix.j;
        return ix;
    }
    ix.m = unit % p.Nm;
    int r = unit / p.Nm;
    const int zi = r % p.ZG; r /= p.ZG;
    ix.j = r % p.J; r /= p.J;
    ix.z = (r % (p.Nz / p.ZG)) * p.ZG + zi;
    ix.s = r / (p.Nz / p.ZG);
    ix.szj = (ix.s * p.Nz + ix.z) * p.J + ix.j;
    return ix;
}

template <class C, class SY, int MODE>
__device__ __forceinline__ void bracket_row_unit(const NlParams& p, const int unit, float2* __restrict__ W,
                                                 float2* __restrict__ S, const float2* __restrict__ twx,
                                                 unsigned long long* stage_bar, float* Tsh, const SY sy) {
    constexpr int NX = C::NX, NY = C::NY, NK = C::NKP;      // NK: plane stride of g, bhat, out in memory
    const int tid = sy.tid();
    constexpr bool CHAIN = MODE != 0;
    const UnitIdx ix = decode_unit<MODE>(p, unit);
    const int s = ix.s, m = ix.m, z = ix.z, j = ix.j, szj = ix.szj;
    const size_t lstride = (size_t)p.Nz * NK;
    const float2* __restrict__ g0 = p.g + ((size_t)(s * p.Nm + m) * p.Nl * p.Nz + z) * NK;

    unsigned bar_parity = 0;
    GX_CTA(0);
    GX_CTA(7);
    // The next grid in the stream may be scheduled as soon as every CTA of this one has started: the separate
    // inverse-Laguerre grid (waits on the arrival counters) or, in chained calls, the chi grid of the NEXT call
    // (reuse of dchi / bhat / out is ordered by the counters below, not by grid completion).
    pdl_launch_dependents();
    __shared__ unsigned slot_seen;                    // (kept in shared memory: no register lives across the row phase)
    if (CHAIN && p.done && p.a8_target != 0u && tid == 0) {    // requested now, looked at before x_forward (latency hidden)
        unsigned c;
        asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(c) : "l"(p.count + (s * p.Nm + m) * p.Nz + z) : "memory");
        slot_seen = c;
    }
    unsigned chi_seen = 0;
    if (CHAIN && p.done && tid == 0)                           // same for the flag of this unit's chi plane
        asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(chi_seen) : "l"(p.chi_ready + szj) : "memory");
    if (tid == 0) mbar_init(stage_bar, 1);
    if (tid < p.Nl) Tsh[tid] = __ldg(p.T + j * p.Nl + tid);
    sy.sync();
    // ---- a2: forward Laguerre transform l -> node j, fused into the TMA-staged load
    stage_combine_tma<C, SY>(W, S, stage_bar, bar_parity, g0, lstride, Tsh, p.Nl, sy);
    sy.sync();
    GX_CTA(1);
    // ---- a3 + a4 (x part).  Chained calls whose chi plane was already complete when this unit started (every unit
    // but those of the first wave): the chi rows of the first two output groups are requested into L1 between the
    // two x passes -- an L2 round trip takes about 1 us under this kernel's load, the row phase would otherwise
    // start with it
    const float2* dchi = p.dchi + (size_t)szj * NX * NY;
    __shared__ unsigned chi_early;
    if (tid == 0) chi_early = (CHAIN && p.done && chi_seen == p.chi_epoch) ? 1u : 0u;
    auto early_prefetch = [&]() {
        if (CHAIN && chi_early) {
            for (int row = tid; row < NX; row += C::NT) {
#pragma unroll
                for (int k2 = 0; k2 < 8; ++k2) {
                    asm volatile("prefetch.global.L1 [%0];" ::"l"(dchi + row + (8 * k2) * NX));
                    asm volatile("prefetch.global.L1 [%0];" ::"l"(dchi + row + (1 + 8 * k2) * NX));
                }
            }
        }
    };
    x_inverse<C, false, SY, decltype(early_prefetch)>(W, twx, p.dkx, p.dky, S, sy, early_prefetch);
    GX_CTA(2);

    if (!CHAIN || !p.done) pdl_wait();        // chi planes of this call are complete and visible from here on
    else {
        // chained: every chi CTA of this call is resident (this grid is scheduled after all of them have started);
        // wait for this unit's own plane only
        if (tid == 0) {
            unsigned c = chi_seen;
            while (c != p.chi_epoch) {
                __nanosleep(100);
                asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(c) : "l"(p.chi_ready + szj) : "memory");
            }
        }
        sy.sync();
    }
    GX_CTA(3);
    // ---- a4 (y part) + a5 + a6 (y part) + a7 (ky), one x row per thread, all in registers
    for (int row = tid; row < NX; row += C::NT) {
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
    sy.sync();
    GX_CTA(4);
    // the row phase needs every register: nothing but blockIdx is carried across it, the indices are formed again
    int unit2 = unit;
    if (CHAIN) asm volatile("" : "+r"(unit2));
    const UnitIdx iy = CHAIN ? decode_unit<MODE>(p, unit2) : ix;
    unsigned* cnt = p.count + (iy.s * p.Nm + iy.m) * p.Nz + iy.z;
    if (CHAIN && p.done && tid == 0) {
        atomicAdd(p.done, 1u);          // this unit has read its chi pairs (values consumed before the barrier above)
        if (p.a8_target != 0u) {
            // chained calls: the previous call's closer of this (s,m,z) must have read the bhat slots (and written
            // out) before this call overwrites them; its last action is the arrival that completes count
            unsigned c = slot_seen;
            while ((int)(c - (p.a8_target - (unsigned)p.J)) < 0) {
                __nanosleep(100);
                asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(c) : "l"(cnt) : "memory");
            }
        }
    }
    if constexpr (MODE == 2) {
        // ---- a6 (x part) + a7 into this CTA's S region, then a8 over the cluster's distributed shared memory
        using StoreC = typename std::conditional<C::TR, TrStore<C>, LinearStore>::type;
        x_forward<C, SY, StoreC>(W, twx, S, p.scale, sy);
        GX_CTA(5);
        cluster_sync_all();            // every node plane of this (s,m,z) is complete and visible cluster-wide
        cluster_laguerre_inverse<C, SY>(S, p.out + (((size_t)(iy.s * p.Nm + iy.m) * p.Nl) * p.Nz + iy.z) * NK, (size_t)p.Nz * NK,
                                        p.Tinv, p.J, p.Nl, cluster_ctarank(), sy);
        cluster_sync_all();            // nobody leaves while its plane is still being read; all of out is written
        if (tid == 0 && iy.j == 0) arrive_release_n(cnt, (unsigned)p.J);     // completes the epoch (+J per call)
        GX_CTA(6);
        return;
    }
    // ---- a6 (x part) + a7 (keep |kx| <= K)
    using Store = typename std::conditional<C::TR, TrStore<C>, LinearStore>::type;
    x_forward<C, SY, Store>(W, twx, p.bhat + ((size_t)iy.szj * p.Nm + iy.m) * NK, p.scale, sy);

    // ---- publish (see bracket_kernel)
    sy.sync();
    GX_CTA(5);
    if (MODE == 1 && p.a8_target != 0u && iy.j == p.J - 1) {
        // ---- a8: this unit closes its (s,m,z); its own plane is read back with the others
        closer_sum<C, SY>(W, p.bhat + ((size_t)((iy.s * p.Nz + iy.z) * p.J) * p.Nm + iy.m) * NK, (size_t)p.Nm * NK,
                          p.out + (((size_t)(iy.s * p.Nm + iy.m) * p.Nl) * p.Nz + iy.z) * NK, (size_t)p.Nz * NK, p.Tinv, p.J, p.Nl,
                          cnt, p.a8_target - 1u, stage_bar, bar_parity, sy, p);
        sy.sync();
        if (tid == 0) arrive_release(cnt);     // completes the epoch (+J per call): out is written, bhat read
        GX_CTA(6);
        return;
    }
    if (tid == 0) arrive_release(cnt);
    GX_CTA(6);
}

// CHAIN = false: the plain kernel (separate inverse-Laguerre grid, grid-completion order); CHAIN = true adds the
// closer (a8 in the last node unit) and the counter-ordered chaining of consecutive calls.  Two instantiations: the
// extra code paths cost registers in the row phase (57.5 -> 60-63 us for the Cyclone plane when compiled in).
// (MODE 2: the chained kernel with the cluster epilogue instead of the closer; launched with cluster dimension J.)
template <class C, int MODE>
__global__ void __launch_bounds__(C::NT, C::MINB) bracket_row_kernel(const NlParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2* W = reinterpret_cast<float2*>(smem_raw);
    float2* S = W + C::W_ELEMS;
    float2* twx = S + C::S_ELEMS;
    __shared__ unsigned long long stage_bar;
    __shared__ float Tsh[16];
    for (int i = threadIdx.x; i < C::NX; i += C::NT) twx[i] = p.twx[i];
    bracket_row_unit<C, CtaSync, MODE>(p, blockIdx.x, W, S, twx, &stage_bar, Tsh, CtaSync());
}

}  // namespace gx
