// linear_kernels.cuh -- quasineutrality field solve and the linear terms of Eq. 4.9 (PAPER.md lines
// 212-260, 284, 298-318, 391) for gx_field_solve / gx_linear_rhs / gx_rhs.  SURVEY.md row f1.
//
// Tables are built on the host in fp64 and rounded once to fp32:
//   Jl[s][l][z][k]   = (1/l!)(-b_s/2)^l e^{-b_s/2}           Eq. 4.7 (line 202)
//   invD[z][k]       = 1 / ( sum_s Z^2 n/tau (1 - sum_l Jl^2) [+ Z^2 n/tau * tau_fac if adiabatic] )
//   fsfac[kx]        = pref*tau_fac / (1 - pref*tau_fac <<1/D>>)   (flux-surface-average closure, ky = 0)
#pragma once
#include <cuda_runtime.h>

#include "dft_regs.cuh"

#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

namespace gx {

struct LinSpecies { double Z, mass, temp, dens, tprim, fprim, nu; };

struct LinHostInput {
    int Nz, Nl, Nm, Ns, nakx, naky;
    double dkx, dky, shat, gradpar;
    const double *kp2, *bmag, *gbdrift, *gbdrift0, *cvdrift, *cvdrift0, *bgrad, *jacobian;
    bool adiabatic;
    double tau_fac, D_hyper, f_hyp;
    int n_hyper;
    bool linked = false;       // twist-and-shift linked z operators (Eq. 4.29) instead of periodic per mode
    double damp_A = 0.0, damp_width = 0.125;   // wave-absorbing end layer, Eq. 4.30 (A = 0: off)
    std::vector<LinSpecies> species;
};

constexpr int kMaxSpecies = 4;

struct LinTables {
    int Nz = 0, Nl = 0, Nm = 0, Ns = 0, nakx = 0, naky = 0, nk = 0;
    bool adiabatic = false;
    float* Jl = nullptr;       // [s][l][z][k]
    float* invD = nullptr;     // [z][k]
    float* fsfac = nullptr;    // [kx]
    float* wz = nullptr;       // [z] jacobian weights, sum 1
    float* bs = nullptr;       // [s][z][k]  b_s
    float* Dz = nullptr;       // [Nz] circulant column of gradpar * spectral d/dz:  D[z][z'] = Dz[(z - z') mod Nz]
    float* Az = nullptr;       // [Nz] circulant column of |gradpar| * spectral |k_z|
    float2* twz = nullptr;     // [Nz] e^{+2 pi i t/Nz}: twiddles of the z FFT path (Nz = 64, 96, 128)
    float gradpar = 0.f;
    float* omd = nullptr;      // [2][z][k]  omega_d^kappa, omega_d^gradB
    float* hypv = nullptr;     // [z][k] D (kperp2/kperp2max)^n
    float* dend = nullptr;     // [z][k] end-damping profile d(z_hat) of Eq. 4.30 (nullptr: layer off)
    float* bgrad = nullptr;    // [z]
    float qn[kMaxSpecies] = {0}, zt[kMaxSpecies] = {0}, vt[kMaxSpecies] = {0}, tz[kMaxSpecies] = {0};
    float tprim[kMaxSpecies] = {0}, fprim[kMaxSpecies] = {0}, nu[kMaxSpecies] = {0}, nuhyp[kMaxSpecies] = {0};
    float* mpow = nullptr;     // [Nm] m^p, p = Nm/2 (Eq. 4.27)
    // twist-and-shift linking (Eq. 4.29): chains of compact modes forming one periodic extended domain
    bool linked = false;
    int nchain = 0, max_ext = 0;   // number of chains, longest extended domain in points (L * Nz)
    int* chain_off = nullptr;      // [nchain + 1] offsets into chain_mode
    int* chain_mode = nullptr;     // compact mode index k = kx_row * naky + ky, in order of increasing ballooning angle
    int* ext_off = nullptr;        // [nchain] offset of the chain's circulant columns in ext_d / ext_a
    int* zwork = nullptr;          // [nzwork] (chain << 8 | slice): slices of kZlinkSlice outputs, longest chains first
    int nzwork = 0, nzwork_long = 0, short_ext = 0;   // items [0, nzwork_long) have more than short_ext points
    int* zlong = nullptr;          // [nzlong] chains with more than short_ext points, longest first (lin_zlink_spectral_kernel)
    int nzlong = 0;
    float* ext_d = nullptr;        // per distinct length L: column of gradpar * d/dzeta, L*Nz entries
    float* ext_a = nullptr;        // per distinct length L: column of |gradpar| * |k_zeta|
    float2* mom = nullptr;     // [s][3][z][k] workspace: u_par, u_perp, T of the Dougherty operator
    float dky = 0;
    bool any_nu = false;
    bool built = false;
};

constexpr int kZlinkThreads = 64, kZlinkSlice = 4 * kZlinkThreads;   // outputs per block of lin_zlink_kernel
constexpr int kLinLaunchesFieldSolve = 2;
constexpr int kLinLaunchesRhs = 3;

inline void lin_tables_free(LinTables& t) {
    cudaFree(t.Jl); cudaFree(t.invD); cudaFree(t.fsfac); cudaFree(t.wz); cudaFree(t.bs);
    cudaFree(t.Dz); cudaFree(t.Az); cudaFree(t.twz); cudaFree(t.omd); cudaFree(t.hypv); cudaFree(t.dend); cudaFree(t.bgrad);
    cudaFree(t.mpow); cudaFree(t.mom);
    cudaFree(t.chain_off); cudaFree(t.chain_mode); cudaFree(t.ext_off); cudaFree(t.ext_d); cudaFree(t.ext_a); cudaFree(t.zwork); cudaFree(t.zlong);
    t = LinTables();
}

template <class T>
inline bool lin_upload(T** dst, const std::vector<T>& src, size_t& bytes, std::string& msg) {
    if (*dst) cudaFree(*dst);
    *dst = nullptr;
    cudaError_t e = cudaMalloc((void**)dst, src.size() * sizeof(T));
    if (e == cudaSuccess) e = cudaMemcpy(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { msg = std::string("linear tables: ") + cudaGetErrorString(e); return false; }
    bytes += src.size() * sizeof(T);
    return true;
}

inline bool lin_tables_build(const LinHostInput& in, LinTables& t, size_t& bytes, std::string& msg) {
    if ((int)in.species.size() > kMaxSpecies) { msg = "at most 4 species"; return false; }
    if ((double)in.Ns * in.Nm * in.Nl * in.Nz * in.nakx * in.naky >= 2147483648.0) {
        msg = "linear kernels index the state with 32 bits: more than 2^31 coefficients";
        return false;
    }
    const int Nz = in.Nz, Nl = in.Nl, Ns = in.Ns, nakx = in.nakx, naky = in.naky;
    const size_t nk = (size_t)nakx * naky;
    const int K = (nakx - 1) / 2;
    t.Nz = Nz; t.Nl = Nl; t.Nm = in.Nm; t.Ns = Ns; t.nakx = nakx; t.naky = naky; t.nk = (int)nk;
    t.adiabatic = in.adiabatic;
    t.dky = (float)in.dky;

    std::vector<float> Jl((size_t)Ns * Nl * Nz * nk), bs((size_t)Ns * Nz * nk);
    std::vector<double> den((size_t)Nz * nk, 0.0);
    for (int s = 0; s < Ns; ++s) {
        const LinSpecies& sp = in.species[s];
        const double rho2 = sp.temp * sp.mass / (sp.Z * sp.Z);
        t.qn[s] = (float)(sp.Z * sp.dens);
        t.zt[s] = (float)(sp.Z / sp.temp);
        t.tz[s] = (float)(sp.temp / sp.Z);
        t.vt[s] = (float)std::sqrt(sp.temp / sp.mass);
        t.tprim[s] = (float)sp.tprim; t.fprim[s] = (float)sp.fprim; t.nu[s] = (float)sp.nu;
        for (int z = 0; z < Nz; ++z)
            for (size_t k = 0; k < nk; ++k) {
                const double b = in.kp2[(size_t)z * nk + k] * rho2 / (in.bmag[z] * in.bmag[z]);
                bs[((size_t)s * Nz + z) * nk + k] = (float)b;
                double jl = std::exp(-0.5 * b), g0 = 0.0;
                for (int l = 0; l < Nl; ++l) {
                    Jl[(((size_t)s * Nl + l) * Nz + z) * nk + k] = (float)jl;
                    g0 += jl * jl;
                    jl *= (-0.5 * b) / (l + 1);
                }
                den[(size_t)z * nk + k] += sp.Z * sp.Z * sp.dens / sp.temp * (1.0 - g0);
            }
    }
    std::vector<float> invD((size_t)Nz * nk), fsfac(nakx, 0.f), wz(Nz);
    double jsum = 0;
    for (int z = 0; z < Nz; ++z) jsum += in.jacobian[z];
    for (int z = 0; z < Nz; ++z) wz[z] = (float)(in.jacobian[z] / jsum);
    const double pref = in.species[0].Z * in.species[0].Z * in.species[0].dens / in.species[0].temp;
    for (size_t i = 0; i < den.size(); ++i) {
        const double D = den[i] + (in.adiabatic ? pref * in.tau_fac : 0.0);
        invD[i] = D != 0.0 ? (float)(1.0 / D) : 0.f;
    }
    if (in.adiabatic) {
        for (int i = 0; i < nakx; ++i) {
            double avg = 0;
            for (int z = 0; z < Nz; ++z)
                avg += in.jacobian[z] / jsum / (den[((size_t)z * nakx + i) * naky] + pref * in.tau_fac);
            const double d = 1.0 - pref * in.tau_fac * avg;
            fsfac[i] = (i == 0 || d == 0.0) ? 0.f : (float)(pref * in.tau_fac / d);
        }
    }
    // ---- linear-term tables (Eq. 4.9-4.18, 4.26-4.28; readings L2-L6 of DESIGN.md)
    std::vector<float> omd(2 * (size_t)Nz * nk), hypv((size_t)Nz * nk), bgr(Nz), dzc(Nz), azc(Nz), mpow(in.Nm);
    double kp2max = 0;
    for (size_t i = 0; i < (size_t)Nz * nk; ++i) kp2max = std::max(kp2max, in.kp2[i]);
    for (int z = 0; z < Nz; ++z) {
        bgr[z] = (float)in.bgrad[z];
        for (int i = 0; i < nakx; ++i) {
            const double kx = in.dkx * (i <= K ? i : i - nakx);
            for (int q = 0; q < naky; ++q) {
                const double ky = in.dky * q;
                const size_t k = ((size_t)z * nakx + i) * naky + q;
                omd[k] = (float)(0.5 * (ky * in.cvdrift[z] + kx * in.cvdrift0[z] / in.shat));
                omd[(size_t)Nz * nk + k] = (float)(0.5 * (ky * in.gbdrift[z] + kx * in.gbdrift0[z] / in.shat));
                hypv[k] = kp2max > 0 ? (float)(in.D_hyper * std::pow(in.kp2[k] / kp2max, (double)in.n_hyper)) : 0.f;
            }
        }
    }
    for (int d = 0; d < Nz; ++d) {
        double sd = 0, sa = 0;
        for (int kk = 0; kk < Nz; ++kk) {
            const int kz = kk <= Nz / 2 ? kk : kk - Nz;
            const double ang = 2.0 * M_PI * (double)kz * d / Nz;
            if (!(Nz % 2 == 0 && kk == Nz / 2)) sd -= kz * std::sin(ang);   // Nyquist dropped in d/dz
            sa += std::abs((double)kz) * std::cos(ang);
        }
        dzc[d] = (float)(in.gradpar * sd / Nz);
        azc[d] = (float)(std::abs(in.gradpar) * sa / Nz);
    }
    {
        std::vector<float2> tw(Nz);
        for (int i = 0; i < Nz; ++i) tw[i] = make_float2((float)std::cos(2.0 * M_PI * i / Nz), (float)std::sin(2.0 * M_PI * i / Nz));
        if (!lin_upload(&t.twz, tw, bytes, msg)) return false;
        t.gradpar = (float)in.gradpar;
    }
    const double p_hyp = 0.5 * in.Nm, m_max = std::max(in.Nm - 1, 1);
    for (int m = 0; m < in.Nm; ++m) mpow[m] = m > 2 ? (float)std::pow((double)m, p_hyp) : 0.f;
    t.any_nu = false;
    for (int s = 0; s < Ns; ++s) {
        t.nuhyp[s] = (float)(2.5 * in.f_hyp * (p_hyp + 0.5) / std::pow(m_max, p_hyp + 0.5) * std::sqrt(in.species[s].temp / in.species[s].mass));
        if (in.species[s].nu != 0.0) t.any_nu = true;
    }
    if (!lin_upload(&t.omd, omd, bytes, msg) || !lin_upload(&t.hypv, hypv, bytes, msg) ||
        !lin_upload(&t.bgrad, bgr, bytes, msg) || !lin_upload(&t.Dz, dzc, bytes, msg) ||
        !lin_upload(&t.Az, azc, bytes, msg) || !lin_upload(&t.mpow, mpow, bytes, msg))
        return false;
    {
        std::vector<float2> zero((size_t)Ns * 3 * Nz * nk, make_float2(0.f, 0.f));
        if (!lin_upload(&t.mom, zero, bytes, msg)) return false;
    }
    t.linked = in.linked;
    if (in.linked) {
        const double jt = 2.0 * M_PI * in.shat * in.dky / in.dkx;
        const int jtw = (int)std::lround(jt);
        if (std::abs(jt - jtw) > 1e-6 || jtw == 0) { msg = "box is not twist-shift quantised: 2 pi shat dky/dkx is not a non-zero integer"; return false; }
        std::vector<int> coff{0}, cmode, eoff;
        std::vector<int> len_off(nakx + 2, -1);
        std::vector<float> ed, ea;
        int max_ext = 0;
        auto row_of = [&](int pidx) { return pidx >= 0 ? pidx : pidx + nakx; };
        for (int q = 0; q < naky; ++q) {
            const int step = jtw * q;
            for (int pidx = -K; pidx <= K; ++pidx) {
                std::vector<int> members;
                if (step == 0) members.push_back(pidx);
                else {
                    if (std::abs(pidx - step) <= K) continue;            // has a predecessor in the dealiased set
                    for (int pp = pidx; std::abs(pp) <= K; pp += step) members.push_back(pp);
                }
                const int L = (int)members.size();
                // mode n holds theta = z - 2 pi n: increasing ballooning angle runs n = L-1, ..., 0
                for (int n = L - 1; n >= 0; --n) cmode.push_back(row_of(members[n]) * naky + q);
                coff.push_back((int)cmode.size());
                if (len_off[L] < 0) {
                    len_off[L] = (int)ed.size();
                    const int N = L * Nz;
                    for (int d = 0; d < N; ++d) {
                        double sd = 0, sa = 0;
                        for (int jj = 0; jj < N; ++jj) {
                            const int j = jj <= N / 2 ? jj : jj - N;
                            const double ang = 2.0 * M_PI * (double)j * d / N;
                            if (!(N % 2 == 0 && jj == N / 2)) sd -= ((double)j / L) * std::sin(ang);
                            sa += (std::abs((double)j) / L) * std::cos(ang);
                        }
                        ed.push_back((float)(in.gradpar * sd / N));
                        ea.push_back((float)(std::abs(in.gradpar) * sa / N));
                    }
                }
                eoff.push_back(len_off[L]);
                max_ext = std::max(max_ext, L * Nz);
            }
        }
        t.nchain = (int)eoff.size();
        t.max_ext = max_ext;
        std::vector<int> order(t.nchain), work;
        for (int c = 0; c < t.nchain; ++c) order[c] = c;
        std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return coff[a + 1] - coff[a] > coff[b + 1] - coff[b]; });
        for (int c : order) {
            const int N = (coff[c + 1] - coff[c]) * Nz;
            for (int sl = 0; sl * kZlinkSlice < N; ++sl) work.push_back((c << 8) | sl);
        }
        t.nzwork = (int)work.size();
        t.short_ext = std::min(max_ext, 4 * Nz);
        t.nzwork_long = 0;
        for (int w : work)
            if ((coff[(w >> 8) + 1] - coff[w >> 8]) * Nz > t.short_ext) t.nzwork_long++;
        if (max_ext > 255 * kZlinkSlice) { msg = "extended domain too long for the slice encoding"; return false; }
        if (!lin_upload(&t.zwork, work, bytes, msg)) return false;
        std::vector<int> zlong;
        for (int c : order)
            if ((coff[c + 1] - coff[c]) * Nz > t.short_ext) zlong.push_back(c);
        t.nzlong = (int)zlong.size();
        if (t.nzlong > 0 && !lin_upload(&t.zlong, zlong, bytes, msg)) return false;
        if (!lin_upload(&t.chain_off, coff, bytes, msg) || !lin_upload(&t.chain_mode, cmode, bytes, msg) ||
            !lin_upload(&t.ext_off, eoff, bytes, msg) || !lin_upload(&t.ext_d, ed, bytes, msg) ||
            !lin_upload(&t.ext_a, ea, bytes, msg))
            return false;
    }
    // ---- wave-absorbing layer at the ends of every extended z domain, Eq. 4.30: d = A [1 - 2 zh^2/(1 + zh^4)]
    // for |zh| < 1, zh = distance from either end / (damp_width * L_z), L_z = 2 pi L; ky = 0 untouched (reading L9)
    if (t.dend) { cudaFree(t.dend); t.dend = nullptr; }
    if (in.damp_A != 0.0) {
        std::vector<float> dend((size_t)Nz * nk, 0.f);
        const double jt = 2.0 * M_PI * in.shat * in.dky / in.dkx;
        const int jtw = in.linked ? (int)std::lround(jt) : 0;
        for (int q = 1; q < naky; ++q) {
            const int step = jtw * q;
            for (int pidx = -K; pidx <= K; ++pidx) {
                std::vector<int> members;
                if (step == 0) members.push_back(pidx);
                else {
                    if (std::abs(pidx - step) <= K) continue;
                    for (int pp = pidx; std::abs(pp) <= K; pp += step) members.push_back(pp);
                }
                const int L = (int)members.size();
                const double w = in.damp_width * 2.0 * M_PI * L, lo = -M_PI - 2.0 * M_PI * (L - 1), hi = M_PI;
                for (int n = 0; n < L; ++n) {
                    const int row = members[n] >= 0 ? members[n] : members[n] + nakx;
                    for (int z = 0; z < Nz; ++z) {
                        const double theta = -M_PI + 2.0 * M_PI * z / Nz - 2.0 * M_PI * n;
                        double d = 0.0;
                        for (double dist : {theta - lo, hi - theta}) {
                            const double zh = dist / w;
                            if (zh < 1.0) d += in.damp_A * (1.0 - 2.0 * zh * zh / (1.0 + zh * zh * zh * zh));
                        }
                        dend[((size_t)z * nakx + row) * naky + q] = (float)d;
                    }
                }
            }
        }
        if (!lin_upload(&t.dend, dend, bytes, msg)) return false;
    }
    if (!lin_upload(&t.Jl, Jl, bytes, msg) || !lin_upload(&t.bs, bs, bytes, msg) ||
        !lin_upload(&t.invD, invD, bytes, msg) || !lin_upload(&t.fsfac, fsfac, bytes, msg) ||
        !lin_upload(&t.wz, wz, bytes, msg))
        return false;
    t.built = true;
    return true;
}

// phi_raw[z][k] = invD * sum_s Z n sum_l Jl G[s,0,l,z,k];  phi(0,0) = 0
__global__ void __launch_bounds__(256) field_solve_kernel(LinTables t, const float2* __restrict__ g,
                                                          float2* __restrict__ phi) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    const int z = blockIdx.y;
    if (k >= t.nk) return;
    float2 num = make_float2(0.f, 0.f);
    for (int s = 0; s < t.Ns; ++s) {
        float2 nb = make_float2(0.f, 0.f);
        for (int l = 0; l < t.Nl; ++l) {
            const float j = t.Jl[(((size_t)s * t.Nl + l) * t.Nz + z) * t.nk + k];
            const float2 f = g[((((size_t)s * t.Nm + 0) * t.Nl + l) * t.Nz + z) * t.nk + k];
            nb.x = fmaf(j, f.x, nb.x);
            nb.y = fmaf(j, f.y, nb.y);
        }
        num.x = fmaf(t.qn[s], nb.x, num.x);
        num.y = fmaf(t.qn[s], nb.y, num.y);
    }
    const float d = t.invD[(size_t)z * t.nk + k];
    phi[(size_t)z * t.nk + k] = (k == 0) ? make_float2(0.f, 0.f) : make_float2(num.x * d, num.y * d);
}

// adiabatic electrons, ky = 0 rows: phi += fsfac[kx] * <<phi_raw>>_z * invD   (Eq. 6.1 solved for <<phi>>).
// One warp per kx row; lanes stride over z and reduce by shuffle.
__global__ void __launch_bounds__(32) flux_surface_kernel(LinTables t, float2* __restrict__ phi) {
    const int i = blockIdx.x + 1;                           // kx row; row 0 (kx = 0) keeps phi(0,0) = 0
    if (i >= t.nakx) return;
    const size_t col = (size_t)i * t.naky;
    float2 avg = make_float2(0.f, 0.f);
    for (int z = threadIdx.x; z < t.Nz; z += 32) {
        const float2 f = phi[(size_t)z * t.nk + col];
        avg.x = fmaf(t.wz[z], f.x, avg.x);
        avg.y = fmaf(t.wz[z], f.y, avg.y);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        avg.x += __shfl_xor_sync(0xffffffffu, avg.x, o);
        avg.y += __shfl_xor_sync(0xffffffffu, avg.y, o);
    }
    const float fs = t.fsfac[i];
    for (int z = threadIdx.x; z < t.Nz; z += 32) {
        const float d = t.invD[(size_t)z * t.nk + col] * fs;
        float2 f = phi[(size_t)z * t.nk + col];
        f.x = fmaf(d, avg.x, f.x);
        f.y = fmaf(d, avg.y, f.y);
        phi[(size_t)z * t.nk + col] = f;
    }
}

inline cudaError_t lin_field_solve(const LinTables& t, const float2* g, float2* phi, cudaStream_t st) {
    if (!t.built) return cudaErrorNotReady;
    dim3 grid((t.nk + 255) / 256, t.Nz);
    field_solve_kernel<<<grid, 256, 0, st>>>(t, g, phi);
    if (t.adiabatic && t.nakx > 1) flux_surface_kernel<<<t.nakx - 1, 32, 0, st>>>(t, phi);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Electromagnetic field solve, Eq. 4.23-4.25: per (z,k) a 2x2 system for (Phi, dB_par/B)
// and the decoupled parallel Ampere law for A_par; kinetic species only; fields vanish at kx = ky = 0.
struct EmSpecies { float qn[kMaxSpecies], z2nt[kMaxSpecies], nt[kMaxSpecies], z2nm[kMaxSpecies], qnv[kMaxSpecies]; };
__global__ void __launch_bounds__(256) field_solve_em_kernel(LinTables t, EmSpecies e, const float* __restrict__ kp2,
                                                             const float* __restrict__ bmag2, float beta,
                                                             const float2* __restrict__ g, float2* __restrict__ phi,
                                                             float2* __restrict__ apar, float2* __restrict__ bpar) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    const int z = blockIdx.y;
    if (k >= t.nk) return;
    float a11 = 0.f, a12 = 0.f, a22 = 0.f, amp = 0.f;
    float2 r1 = make_float2(0.f, 0.f), r2 = r1, ra = r1;
    for (int s = 0; s < t.Ns; ++s) {
        float sjj = 0.f, sjb = 0.f, sbb = 0.f, jprev = 0.f;
        float2 n0 = make_float2(0.f, 0.f), nb = n0, n1 = n0;
        for (int l = 0; l < t.Nl; ++l) {
            const float j = t.Jl[(((size_t)s * t.Nl + l) * t.Nz + z) * t.nk + k], jb = j + jprev;
            jprev = j;
            sjj = fmaf(j, j, sjj); sjb = fmaf(j, jb, sjb); sbb = fmaf(jb, jb, sbb);
            const float2 g0 = g[((((size_t)s * t.Nm + 0) * t.Nl + l) * t.Nz + z) * t.nk + k];
            n0.x = fmaf(j, g0.x, n0.x); n0.y = fmaf(j, g0.y, n0.y);
            nb.x = fmaf(jb, g0.x, nb.x); nb.y = fmaf(jb, g0.y, nb.y);
            if (t.Nm > 1) {
                const float2 g1 = g[((((size_t)s * t.Nm + 1) * t.Nl + l) * t.Nz + z) * t.nk + k];
                n1.x = fmaf(j, g1.x, n1.x); n1.y = fmaf(j, g1.y, n1.y);
            }
        }
        a11 += e.z2nt[s] * (1.f - sjj);
        a12 += e.qn[s] * sjb;
        a22 += e.nt[s] * sbb;
        amp += e.z2nm[s] * sjj;
        r1.x = fmaf(e.qn[s], n0.x, r1.x); r1.y = fmaf(e.qn[s], n0.y, r1.y);
        r2.x = fmaf(e.nt[s], nb.x, r2.x); r2.y = fmaf(e.nt[s], nb.y, r2.y);
        ra.x = fmaf(e.qnv[s], n1.x, ra.x); ra.y = fmaf(e.qnv[s], n1.y, ra.y);
    }
    const float h = 0.5f * beta / bmag2[z];
    const float det = a11 * (1.f + h * a22) + a12 * h * a12;
    const float idet = det != 0.f ? 1.f / det : 0.f;
    const float c11 = (1.f + h * a22) * idet, c12 = -a12 * h * idet, c21 = -h * a12 * idet, c22 = -a11 * h * idet;
    const float den = kp2[(size_t)z * t.nk + k] + 0.5f * beta * amp;
    const float ia = den != 0.f ? 0.5f * beta / den : 0.f;
    const size_t o = (size_t)z * t.nk + k;
    const bool zero = k == 0;
    phi[o] = zero ? make_float2(0.f, 0.f) : make_float2(c11 * r1.x + c12 * r2.x, c11 * r1.y + c12 * r2.y);
    bpar[o] = zero ? make_float2(0.f, 0.f) : make_float2(c21 * r1.x + c22 * r2.x, c21 * r1.y + c22 * r2.y);
    apar[o] = zero ? make_float2(0.f, 0.f) : make_float2(ia * ra.x, ia * ra.y);
}

// chi planes of the electromagnetic brackets in spectral form: chis[unit = (s,z,j)][k] = M fa + MB fb  (fb may be null)
__global__ void __launch_bounds__(256) em_chi_spectral_kernel(const float* __restrict__ M, const float* __restrict__ MB,
                                                              const float2* __restrict__ fa, const float2* __restrict__ fb,
                                                              float2* __restrict__ chis, int nk, int Nz, int J) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    const int unit = blockIdx.y;
    if (k >= nk) return;
    const int z = (unit / J) % Nz;
    const size_t i = (size_t)unit * nk + k;
    const float2 a = fa[(size_t)z * nk + k];
    float2 r = make_float2(M[i] * a.x, M[i] * a.y);
    if (fb) {
        const float2 b = fb[(size_t)z * nk + k];
        r.x = fmaf(MB[i], b.x, r.x);
        r.y = fmaf(MB[i], b.y, r.y);
    }
    chis[i] = r;
}

// g2_{l,m} = -v_ts ( sqrt(m+1) G_{l,m+1} + sqrt(m) G_{l,m-1} )  (Hermite recurrence of v_par; G outside 0 <= m < Nm is 0)
__global__ void __launch_bounds__(256) em_hermite_shift_kernel(LinTables t, const float2* __restrict__ g, float2* __restrict__ g2) {
    const unsigned pl = (unsigned)(t.Nl * t.Nz * t.nk);       // elements of one (s,m) slab
    const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= pl) return;
    const int s = blockIdx.y / t.Nm, m = blockIdx.y % t.Nm;
    const float up = -t.vt[s] * sqrtf((float)(m + 1)), dn = -t.vt[s] * sqrtf((float)m);
    float2 r = make_float2(0.f, 0.f);
    if (m + 1 < t.Nm) { const float2 a = g[(size_t)(s * t.Nm + m + 1) * pl + i]; r.x = up * a.x; r.y = up * a.y; }
    if (m > 0) { const float2 a = g[(size_t)(s * t.Nm + m - 1) * pl + i]; r.x = fmaf(dn, a.x, r.x); r.y = fmaf(dn, a.y, r.y); }
    g2[(size_t)(s * t.Nm + m) * pl + i] = r;
}
__global__ void __launch_bounds__(256) em_add_kernel(float4* __restrict__ out, const float4* __restrict__ add, size_t n4) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n4) { float4 a = out[i]; const float4 b = add[i]; a.x += b.x; a.y += b.y; a.z += b.z; a.w += b.w; out[i] = a; }
}

// ------------------------------------------------------------------------------------------------
// Linear terms of Eq. 4.9 for gx_linear_rhs / gx_rhs.
// H_{l,m} = G_{l,m} + (Z/tau) J_l Phi delta_{m0} (Eq. 4.8) is formed on the fly; H, G, J vanish outside
// 0 <= l < Nl, 0 <= m < Nm.
__device__ __forceinline__ float2 lin_H(const LinTables& t, const float2* __restrict__ g, const float2* __restrict__ phi,
                                        int s, int l, int m, int z, int k) {
    if (l < 0 || l >= t.Nl || m < 0 || m >= t.Nm) return make_float2(0.f, 0.f);
    const unsigned zk = (unsigned)(z * t.nk + k), pl = (unsigned)(t.Nz * t.nk);   // < 2^31 elements (checked at build)
    float2 h = g[(unsigned)((s * t.Nm + m) * t.Nl + l) * pl + zk];
    if (m == 0) {
        const float c = t.zt[s] * t.Jl[(unsigned)(s * t.Nl + l) * pl + zk];
        const float2 f = phi[zk];
        h.x = fmaf(c, f.x, h.x);
        h.y = fmaf(c, f.y, h.y);
    }
    return h;
}
__device__ __forceinline__ float lin_J(const LinTables& t, int s, int l, int z, int k) {
    return (l < 0 || l >= t.Nl) ? 0.f : t.Jl[(unsigned)(s * t.Nl + l) * (unsigned)(t.Nz * t.nk) + (unsigned)(z * t.nk + k)];
}

// field-particle moments of the Dougherty operator, Eq. 4.14-4.18: mom[s][0..2][z][k]
__global__ void __launch_bounds__(256) lin_moments_kernel(LinTables t, const float2* __restrict__ g,
                                                          const float2* __restrict__ phi) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    const int z = blockIdx.y, s = blockIdx.z;
    if (k >= t.nk) return;
    const float b = t.bs[((size_t)s * t.Nz + z) * t.nk + k];
    const float sb = sqrtf(fmaxf(b, 0.f));
    float2 up = make_float2(0.f, 0.f), uq = up, tp = up, tq = up;
    for (int l = 0; l < t.Nl; ++l) {
        const float jm = lin_J(t, s, l - 1, z, k), j0 = lin_J(t, s, l, z, k), jp = lin_J(t, s, l + 1, z, k);
        const float2 h0 = lin_H(t, g, phi, s, l, 0, z, k), h1 = lin_H(t, g, phi, s, l, 1, z, k),
                     h2 = lin_H(t, g, phi, s, l, 2, z, k);
        const float cq = j0 + jm, ct = l * jm + 2.f * l * j0 + (l + 1.f) * jp;
        up.x = fmaf(j0, h1.x, up.x); up.y = fmaf(j0, h1.y, up.y);
        uq.x = fmaf(cq, h0.x, uq.x); uq.y = fmaf(cq, h0.y, uq.y);
        tp.x = fmaf(j0, h2.x, tp.x); tp.y = fmaf(j0, h2.y, tp.y);
        tq.x = fmaf(ct, h0.x, tq.x); tq.y = fmaf(ct, h0.y, tq.y);
    }
    const float r2 = 1.41421356237309504880f;
    float2* __restrict__ mo = t.mom + ((size_t)s * 3 * t.Nz + z) * t.nk + k;
    const size_t st = (size_t)t.Nz * t.nk;
    mo[0] = up;
    mo[st] = make_float2(sb * uq.x, sb * uq.y);
    mo[2 * st] = make_float2((r2 * tp.x + 2.f * tq.x) * (1.f / 3.f), (r2 * tp.y + 2.f * tq.y) * (1.f / 3.f));
}

constexpr int kLinTK = 16;      // k per block
constexpr int kLinZG = 8;       // z groups per block

// Spectral z operators by FFT (Eq. 4.10-4.11) for long field lines: for every column tk of the tile
//     S1[z] <- F^-1[ -v_t gradpar (i k_z) F[S1] - hyp |gradpar| |k_z| F[S2] ](z)      (Nyquist dropped in the derivative)
// with N = A*B two register-radix passes each way through shared memory: the forward transform is decimation in
// time with digit-transposed output (position k1*B + k2 holds k = k1 + A*k2), the inverse the matching decimation
// in frequency that reads that order and ends in natural order (same scheme as the x passes of nl_kernels.cuh).
// S2 is preserved (the hyper-viscosity term reads G_{l,m} from it later); S3 is scratch for its transform.
template <int A, int B>
__device__ __forceinline__ void lin_zfft(float2* __restrict__ S1, const float2* __restrict__ S2, float2* __restrict__ S3,
                                         const float2* __restrict__ tw, float vt_gp, float hyp_gp, bool with_hyp) {
    constexpr int N = A * B, NT = kLinTK * kLinZG;
    // forward pass 1: DFT_A over n1 of z = n1*B + n2, twiddle e^{-2 pi i n2 k1 / N}
    for (int it = threadIdx.x; it < B * kLinTK; it += NT) {
        const int n2 = it / kLinTK, c = it - n2 * kLinTK;
        float2 v[A], u[A];
#pragma unroll
        for (int n1 = 0; n1 < A; ++n1) {
            v[n1] = S1[(n1 * B + n2) * kLinTK + c];
            u[n1] = with_hyp ? S2[(n1 * B + n2) * kLinTK + c] : make_float2(0.f, 0.f);
        }
        dft<A, -1>(v);
        if (with_hyp) dft<A, -1>(u);
#pragma unroll
        for (int k1 = 0; k1 < A; ++k1) {
            const float2 w = tw[(n2 * k1) % N];
            S1[(k1 * B + n2) * kLinTK + c] = k1 == 0 ? v[0] : cmul_conj(v[k1], w);
            if (with_hyp) S3[(k1 * B + n2) * kLinTK + c] = k1 == 0 ? u[0] : cmul_conj(u[k1], w);
        }
    }
    __syncthreads();
    // forward pass 2 + spectral factors + inverse pass 1 (DFT_B over the same B values: the register tile is reused)
    for (int it = threadIdx.x; it < A * kLinTK; it += NT) {
        const int k1 = it / kLinTK, c = it - k1 * kLinTK;
        float2 v[B], u[B];
#pragma unroll
        for (int n2 = 0; n2 < B; ++n2) {
            v[n2] = S1[(k1 * B + n2) * kLinTK + c];
            u[n2] = with_hyp ? S3[(k1 * B + n2) * kLinTK + c] : make_float2(0.f, 0.f);
        }
        dft<B, -1>(v);
        if (with_hyp) dft<B, -1>(u);
#pragma unroll
        for (int k2 = 0; k2 < B; ++k2) {
            const int k = k1 + A * k2;                           // frequency of this value
            const int kz = k <= N / 2 ? k : k - N;
            const float fd = (N % 2 == 0 && k == N / 2) ? 0.f : -vt_gp * (float)kz * (1.f / N);   // -v_t gradpar i k_z / N
            const float fa = -hyp_gp * fabsf((float)kz) * (1.f / N);
            // (i fd) v + fa u
            v[k2] = make_float2(-fd * v[k2].y + fa * u[k2].x, fd * v[k2].x + fa * u[k2].y);
        }
        // inverse pass 1: for a = k1, DFT_B(+) over b = k2 -> d, twiddle e^{+2 pi i a d / N}
        dft<B, +1>(v);
#pragma unroll
        for (int d = 0; d < B; ++d)
            S1[(k1 * B + d) * kLinTK + c] = d == 0 ? v[0] : cmul(v[d], tw[(k1 * d) % N]);
    }
    __syncthreads();
    // inverse pass 2: for each d, DFT_A(+) over a -> cc; z = d + B*cc (natural order)
    for (int it = threadIdx.x; it < B * kLinTK; it += NT) {
        const int d = it / kLinTK, c = it - d * kLinTK;
        float2 v[A];
#pragma unroll
        for (int a = 0; a < A; ++a) v[a] = S1[(a * B + d) * kLinTK + c];
        dft<A, +1>(v);
        // in place: the item's outputs z = d + B*cc occupy exactly the positions a*B + d it has just read
#pragma unroll
        for (int cc = 0; cc < A; ++cc) S1[(d + B * cc) * kLinTK + c] = v[cc];
    }
    __syncthreads();
}

// out[s,m,l,z,k] (+)= linear terms.  Block: one (s,m,l), a tile of kLinTK modes k, all z.  The spectral
// parallel derivative / |k_par| are circulant Nz x Nz products on tiles staged in shared memory.
// ZB = 4: each thread owns blocks of 4 consecutive z and register-blocks the circulant products (one staged
// value and one new weight per term feed 8 FMAs); ZB = 1 when Nz is not a multiple of 4.
// DERIV_ONLY: only the two z-operator terms (streaming, hyper-collisions), added to out; the pointwise terms
// then come from lin_point_kernel.
// FA x FB > 0: the z operators by FFT (lin_zfft, Nz = FA*FB) instead of the O(Nz^2) circulant products.
template <bool ACC, int ZB, bool DERIV_ONLY = false, int FA = 0, int FB = 0>
__global__ void __launch_bounds__(kLinTK * kLinZG) lin_rhs_kernel(LinTables t, const float2* __restrict__ g,
                                                                 const float2* __restrict__ phi,
                                                                 float2* __restrict__ out, const bool skip_z) {
    extern __shared__ __align__(16) unsigned char lin_smem[];
    float2* S1 = reinterpret_cast<float2*>(lin_smem);            // [Nz][TK] sqrt(m+1) H_{l,m+1} + sqrt(m) H_{l,m-1}
    float2* S2 = S1 + (size_t)t.Nz * kLinTK;                     // [Nz][TK] G_{l,m} (hyper-collisions)
    float* dz = reinterpret_cast<float*>(S2 + (size_t)t.Nz * kLinTK);   // [2 Nz] column repeated: no wrap test
    float* az = dz + 2 * t.Nz;
    float2* S3 = reinterpret_cast<float2*>(az + 2 * t.Nz);       // FFT path only: [Nz][TK] scratch
    static_assert(FA == 0 || ZB == 1, "the FFT path writes one z per thread and step");
    const int tk = threadIdx.x % kLinTK, zg = threadIdx.x / kLinTK;
    // (s,m) varies fastest over the grid: the blocks that read the slabs m-1, m, m+1 of one k tile run together and
    // share them through L2 (the state of the large configurations is several times the L2 capacity)
    const int k = blockIdx.z * kLinTK + tk;
    const int l = blockIdx.y;
    const int s = blockIdx.x / t.Nm, m = blockIdx.x % t.Nm;
    const bool live = k < t.nk;
    const float sm1 = sqrtf((float)(m + 1)), sm0 = sqrtf((float)m);
    if constexpr (FA > 0) {
        float2* tws = reinterpret_cast<float2*>(dz);              // [Nz] twiddles in place of the circulant columns
        for (int i = threadIdx.x; i < t.Nz; i += blockDim.x) tws[i] = t.twz[i];
    } else {
        for (int i = threadIdx.x; i < 2 * t.Nz; i += blockDim.x) {
            const int d = i < t.Nz ? i : i - t.Nz;
            dz[i] = t.Dz[d];
            az[i] = t.Az[d];
        }
    }
    {
        // staging: 4 z at a time, every load issued before the first use (indices clamped, invalid masked)
        const unsigned pl = (unsigned)(t.Nz * t.nk);
        const int kc = live ? k : t.nk - 1;
        const bool vp = m + 1 < t.Nm, vm = m - 1 >= 0;
        const unsigned ip = (unsigned)((s * t.Nm + (vp ? m + 1 : m)) * t.Nl + l) * pl,
                       im = (unsigned)((s * t.Nm + (vm ? m - 1 : m)) * t.Nl + l) * pl,
                       i0 = (unsigned)((s * t.Nm + m) * t.Nl + l) * pl, ij = (unsigned)(s * t.Nl + l) * pl;
        const float cp = vp ? sm1 : 0.f, cm = vm ? sm0 : 0.f;
        const float cphi = (vm && m == 1) ? sm0 * t.zt[s] : 0.f;          // H_{l,0} = G_{l,0} + (Z/tau) J_l Phi
        if constexpr (FA > 0) {
            // FFT path (Nz >= 64): the three input planes go to shared memory with cp.async -- all Nz/ZG x 3 requests of
            // a thread in flight at once, no registers held -- and are combined in place afterwards
            constexpr int NZT = FA * FB / kLinZG;
            auto cp8 = [](float2* dst, const float2* src) {
                asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
            };
#pragma unroll
            for (int i = 0; i < NZT; ++i) {
                const int z = zg + i * kLinZG;
                const unsigned zk = (unsigned)(z * t.nk + kc);
                cp8(S1 + z * kLinTK + tk, g + ip + zk);
                cp8(S3 + z * kLinTK + tk, g + im + zk);
                cp8(S2 + z * kLinTK + tk, g + i0 + zk);
            }
            asm volatile("cp.async.commit_group;" ::: "memory");
            asm volatile("cp.async.wait_group 0;" ::: "memory");
#pragma unroll
            for (int i = 0; i < NZT; ++i) {
                const int z = zg + i * kLinZG;
                const float2 a = S1[z * kLinTK + tk], b = S3[z * kLinTK + tk];
                float2 r = make_float2(cp * a.x + cm * b.x, cp * a.y + cm * b.y);
                if (cphi != 0.f) {
                    const unsigned zk = (unsigned)(z * t.nk + kc);
                    const float2 f = phi[zk];
                    const float w = cphi * t.Jl[ij + zk];
                    r.x = fmaf(w, f.x, r.x); r.y = fmaf(w, f.y, r.y);
                }
                S1[z * kLinTK + tk] = live ? r : make_float2(0.f, 0.f);
                if (!live) S2[z * kLinTK + tk] = make_float2(0.f, 0.f);
            }
        } else {
        // (circulant path: four z per thread and round trip; Phi and J_l only where they enter, m = 1)
        constexpr int ZBATCH = 4;
        for (int zb = zg; zb < t.Nz; zb += ZBATCH * kLinZG) {
            float2 a[ZBATCH], b[ZBATCH], c[ZBATCH], f[ZBATCH];
            float jl[ZBATCH];
#pragma unroll
            for (int i = 0; i < ZBATCH; ++i) {
                const int z = min(zb + i * kLinZG, t.Nz - 1);
                const unsigned zk = (unsigned)(z * t.nk + kc);
                a[i] = g[ip + zk]; b[i] = g[im + zk]; c[i] = g[i0 + zk];
                if (cphi != 0.f) { f[i] = phi[zk]; jl[i] = t.Jl[ij + zk]; }
                else { f[i] = make_float2(0.f, 0.f); jl[i] = 0.f; }
            }
#pragma unroll
            for (int i = 0; i < ZBATCH; ++i) {
                const int z = zb + i * kLinZG;
                if (z < t.Nz) {
                    const float w = cphi * jl[i];
                    S1[z * kLinTK + tk] = live ? make_float2(cp * a[i].x + cm * b[i].x + w * f[i].x,
                                                             cp * a[i].y + cm * b[i].y + w * f[i].y)
                                               : make_float2(0.f, 0.f);
                    S2[z * kLinTK + tk] = live ? c[i] : make_float2(0.f, 0.f);
                }
            }
        }
        }
    }
    __syncthreads();
    if constexpr (FA > 0) {
        // every thread of the block takes part (dead columns hold zeros)
        if (!skip_z)
            lin_zfft<FA, FB>(S1, S2, S3, reinterpret_cast<const float2*>(dz), t.vt[s] * t.gradpar,
                             t.nuhyp[s] * t.mpow[m] * fabsf(t.gradpar), t.nuhyp[s] * t.mpow[m] != 0.f);
    }
    if (!live) return;
    if constexpr (DERIV_ONLY && FA > 0) {
        // out += (both z-operator terms): every previous value is requested before the first store -- the generic
        // loop below reads and writes out once per z and the stores keep the next load from being issued early
        // (16 dependent round trips per thread: the kernel ran at a sixth of the DRAM bandwidth)
        constexpr int NZT = FA * FB / kLinZG;
        static_assert(FA * FB % kLinZG == 0, "z per thread");
        float2* __restrict__ o0 = out + ((unsigned)((s * t.Nm + m) * t.Nl + l) * (unsigned)(t.Nz * t.nk) + (unsigned)k);
        float2 prev[NZT];
#pragma unroll
        for (int i = 0; i < NZT; ++i) prev[i] = o0[(unsigned)((zg + i * kLinZG) * t.nk)];
        if (!skip_z) {
#pragma unroll
            for (int i = 0; i < NZT; ++i) {
                const float2 r = S1[(zg + i * kLinZG) * kLinTK + tk];
                o0[(unsigned)((zg + i * kLinZG) * t.nk)] = make_float2(prev[i].x + r.x, prev[i].y + r.y);
            }
        }
        return;
    }
    const float vt = t.vt[s], tz = t.tz[s], nu = t.nu[s];
    const float hyp = t.nuhyp[s] * t.mpow[m];
    const float ky = t.dky * (float)(k % t.naky);
    const float fl = (float)l, fm = (float)m;
    for (int zb = zg; zb * ZB < t.Nz; zb += kLinZG) {
      const int z0 = zb * ZB;
      // streaming: -v_t grad_par(...)   and hyper-collisions: -nu_hyp m^p |k_par| G
      float2 dpb[ZB], apb[ZB];
#pragma unroll
      for (int i = 0; i < ZB; ++i) dpb[i] = apb[i] = make_float2(0.f, 0.f);
      {
          auto blocked = [&](const float* __restrict__ col, const float2* __restrict__ sv, float2 (&acc)[ZB]) {
              const float* __restrict__ dc = col + z0 + t.Nz;          // weight of (z0 + i, zp) = dc[i - zp]
              if constexpr (ZB == 4) {
                  float w0 = dc[0], w1 = dc[1], w2 = dc[2], w3 = dc[3];
                  for (int zp = 0; zp < t.Nz; zp += 4) {
                      const float2 a0 = sv[zp * kLinTK], a1 = sv[(zp + 1) * kLinTK], a2 = sv[(zp + 2) * kLinTK],
                                   a3 = sv[(zp + 3) * kLinTK];
                      const float n0 = dc[-(zp + 1)], n1 = dc[-(zp + 2)], n2 = dc[-(zp + 3)], n3 = dc[-(zp + 4)];
                      acc[0].x = fmaf(w0, a0.x, acc[0].x); acc[0].y = fmaf(w0, a0.y, acc[0].y);
                      acc[1].x = fmaf(w1, a0.x, acc[1].x); acc[1].y = fmaf(w1, a0.y, acc[1].y);
                      acc[2].x = fmaf(w2, a0.x, acc[2].x); acc[2].y = fmaf(w2, a0.y, acc[2].y);
                      acc[3].x = fmaf(w3, a0.x, acc[3].x); acc[3].y = fmaf(w3, a0.y, acc[3].y);
                      acc[0].x = fmaf(n0, a1.x, acc[0].x); acc[0].y = fmaf(n0, a1.y, acc[0].y);
                      acc[1].x = fmaf(w0, a1.x, acc[1].x); acc[1].y = fmaf(w0, a1.y, acc[1].y);
                      acc[2].x = fmaf(w1, a1.x, acc[2].x); acc[2].y = fmaf(w1, a1.y, acc[2].y);
                      acc[3].x = fmaf(w2, a1.x, acc[3].x); acc[3].y = fmaf(w2, a1.y, acc[3].y);
                      acc[0].x = fmaf(n1, a2.x, acc[0].x); acc[0].y = fmaf(n1, a2.y, acc[0].y);
                      acc[1].x = fmaf(n0, a2.x, acc[1].x); acc[1].y = fmaf(n0, a2.y, acc[1].y);
                      acc[2].x = fmaf(w0, a2.x, acc[2].x); acc[2].y = fmaf(w0, a2.y, acc[2].y);
                      acc[3].x = fmaf(w1, a2.x, acc[3].x); acc[3].y = fmaf(w1, a2.y, acc[3].y);
                      acc[0].x = fmaf(n2, a3.x, acc[0].x); acc[0].y = fmaf(n2, a3.y, acc[0].y);
                      acc[1].x = fmaf(n1, a3.x, acc[1].x); acc[1].y = fmaf(n1, a3.y, acc[1].y);
                      acc[2].x = fmaf(n0, a3.x, acc[2].x); acc[2].y = fmaf(n0, a3.y, acc[2].y);
                      acc[3].x = fmaf(w0, a3.x, acc[3].x); acc[3].y = fmaf(w0, a3.y, acc[3].y);
                      w3 = n0; w2 = n1; w1 = n2; w0 = n3;
                  }
              } else {
#pragma unroll 4
                  for (int zp = 0; zp < t.Nz; ++zp) {
                      const float w = dc[-zp];
                      const float2 a = sv[zp * kLinTK];
                      acc[0].x = fmaf(w, a.x, acc[0].x); acc[0].y = fmaf(w, a.y, acc[0].y);
                  }
              }
          };
          if constexpr (FA == 0) {
              if (!skip_z) {                    // linked boundary: the z operators come from lin_zlink_kernel
                  blocked(dz, S1 + tk, dpb);
                  if (hyp != 0.f) blocked(az, S2 + tk, apb);
              }
          }
      }
      // previous values of out for the whole z block before the first store (see the FFT path above)
      float2 prevb[ZB];
      if (ACC || DERIV_ONLY) {
#pragma unroll
          for (int zi = 0; zi < ZB; ++zi)
              prevb[zi] = out[(unsigned)((s * t.Nm + m) * t.Nl + l) * (unsigned)(t.Nz * t.nk) + (unsigned)((z0 + zi) * t.nk + k)];
      }
#pragma unroll
      for (int zi = 0; zi < ZB; ++zi) {
        const int z = z0 + zi;
        const float2 dp = dpb[zi], ap = apb[zi];
        float2 r = make_float2(-vt * dp.x - hyp * ap.x, -vt * dp.y - hyp * ap.y);
        if constexpr (FA > 0) {
            if (!skip_z) r = S1[z * kLinTK + tk];               // both z-operator terms, already scaled (lin_zfft)
        }
        if constexpr (!DERIV_ONLY) {
        const float2 h00 = lin_H(t, g, phi, s, l, m, z, k);
        // mirror force
        {
            const float2 a = lin_H(t, g, phi, s, l, m + 1, z, k), b2 = lin_H(t, g, phi, s, l - 1, m + 1, z, k),
                         c = lin_H(t, g, phi, s, l, m - 1, z, k), d2 = lin_H(t, g, phi, s, l + 1, m - 1, z, k);
            const float ca = -(fl + 1.f) * sm1, cb = -fl * sm1, cc = fl * sm0, cd = (fl + 1.f) * sm0;
            const float f = -vt * t.bgrad[z];
            r.x += f * (ca * a.x + cb * b2.x + cc * c.x + cd * d2.x);
            r.y += f * (ca * a.y + cb * b2.y + cc * c.y + cd * d2.y);
        }
        // curvature and grad-B drifts: -i (tau/Z) w (...)
        {
            const float wk = t.omd[(size_t)z * t.nk + k], wb = t.omd[((size_t)t.Nz + z) * t.nk + k];
            const float2 a = lin_H(t, g, phi, s, l, m + 2, z, k), c = lin_H(t, g, phi, s, l, m - 2, z, k);
            const float2 e = lin_H(t, g, phi, s, l + 1, m, z, k), f2 = lin_H(t, g, phi, s, l - 1, m, z, k);
            const float cA = sqrtf((fm + 1.f) * (fm + 2.f)), cB = 2.f * fm + 1.f, cC = sqrtf(fm * fmaxf(fm - 1.f, 0.f));
            const float bx = wk * (cA * a.x + cB * h00.x + cC * c.x) + wb * ((fl + 1.f) * e.x + (2.f * fl + 1.f) * h00.x + fl * f2.x);
            const float by = wk * (cA * a.y + cB * h00.y + cC * c.y) + wb * ((fl + 1.f) * e.y + (2.f * fl + 1.f) * h00.y + fl * f2.y);
            r.x += tz * by;          // -i (x + i y) = y - i x
            r.y -= tz * bx;
        }
        const float jm = lin_J(t, s, l - 1, z, k), j0 = lin_J(t, s, l, z, k), jp = lin_J(t, s, l + 1, z, k);
        const float jt = fl * jm + 2.f * fl * j0 + (fl + 1.f) * jp;
        // drive (Eq. 4.12, Phi parts): i ky (...) Phi
        if (m == 0 || m == 2) {
            const float2 f = phi[(size_t)z * t.nk + k];
            const float c = m == 0 ? t.fprim[s] * j0 + t.tprim[s] * jt : t.tprim[s] * j0 * 0.70710678118654752440f;
            r.x -= ky * c * f.y;
            r.y += ky * c * f.x;
        }
        // Dougherty collisions (Eq. 4.13)
        if (nu != 0.f) {
            const float b = t.bs[((size_t)s * t.Nz + z) * t.nk + k];
            const float damp = nu * (b + 2.f * fl + fm);
            r.x -= damp * h00.x;
            r.y -= damp * h00.y;
            if (m <= 2) {
                const float2* __restrict__ mo = t.mom + ((size_t)s * 3 * t.Nz + z) * t.nk + k;
                const size_t st = (size_t)t.Nz * t.nk;
                float2 add = make_float2(0.f, 0.f);
                if (m == 0) {
                    const float2 uq = mo[st], tb = mo[2 * st];
                    const float cu = sqrtf(fmaxf(b, 0.f)) * (j0 + jm), ct = 2.f * jt;
                    add = make_float2(cu * uq.x + ct * tb.x, cu * uq.y + ct * tb.y);
                } else if (m == 1) {
                    const float2 up = mo[0];
                    add = make_float2(j0 * up.x, j0 * up.y);
                } else {
                    const float2 tb = mo[2 * st];
                    add = make_float2(1.41421356237309504880f * j0 * tb.x, 1.41421356237309504880f * j0 * tb.y);
                }
                r.x = fmaf(nu, add.x, r.x);
                r.y = fmaf(nu, add.y, r.y);
            }
        }
        // hyper-viscosity (Eq. 4.26)
        {
            const float hv = t.hypv[(size_t)z * t.nk + k];
            const float2 gg = S2[z * kLinTK + tk];
            r.x -= hv * gg.x;
            r.y -= hv * gg.y;
        }
        // wave-absorbing end layer (Eq. 4.30): - d(z_hat) H_{l,m}, non-zonal modes
        if (t.dend) {
            const float dd = t.dend[(size_t)z * t.nk + k];
            r.x -= dd * h00.x;
            r.y -= dd * h00.y;
        }
        }
        float2* __restrict__ o = out + ((unsigned)((s * t.Nm + m) * t.Nl + l) * (unsigned)(t.Nz * t.nk) + (unsigned)(z * t.nk + k));
        if (ACC || DERIV_ONLY) { r.x += prevb[zi].x; r.y += prevb[zi].y; }
        *o = r;
      }
    }
}

// Pointwise terms of Eq. 4.9 (mirror, drifts, drive, Dougherty, hyper-viscosity) for ALL l of one (s,m) at
// one (z,k) per thread: the 5 x Nl stencil values H_{l',m-2..m+2} are loaded once into registers and reused
// by every l (the per-(l,m) kernel above fetches 13 neighbours per output).  Pure streaming, coalesced in k.
template <int MAXL, bool ACC>
__global__ void __launch_bounds__(256) lin_point_kernel(LinTables t, const float2* __restrict__ g,
                                                        const float2* __restrict__ phi, float2* __restrict__ out) {
    const unsigned pl = (unsigned)(t.Nz * t.nk);
    const unsigned zk = blockIdx.y * blockDim.x + threadIdx.x;       // (s,m) fastest over the grid: m-2..m+2 share L2
    if (zk >= pl) return;
    const int s = blockIdx.x / t.Nm, m = blockIdx.x % t.Nm;
    const int z = zk / t.nk, k = zk - z * t.nk;
    const float zt = t.zt[s], vt = t.vt[s], tz = t.tz[s], nu = t.nu[s];
    const float2 f = phi[zk];
    float J[MAXL + 2];                                     // J[l + 1] = J_l, zero outside 0 <= l < Nl
    J[0] = 0.f;
#pragma unroll
    for (int l = 0; l < MAXL; ++l) J[l + 1] = l < t.Nl ? t.Jl[(unsigned)(s * t.Nl + l) * pl + zk] : 0.f;
    J[MAXL + 1] = 0.f;
    // All stencil loads are issued unconditionally (indices clamped, invalid neighbours masked afterwards) so
    // that the 5 x Nl requests are in flight together: the kernel is latency-bound otherwise.
    float2 h[5][MAXL + 2];                                 // h[dm + 2][l + 1] = H_{l, m + dm}
#pragma unroll
    for (int dm = 0; dm < 5; ++dm) {
        const int mm = m + dm - 2;
        const int mc = min(max(mm, 0), t.Nm - 1);
        h[dm][0] = h[dm][MAXL + 1] = make_float2(0.f, 0.f);
#pragma unroll
        for (int l = 0; l < MAXL; ++l)
            h[dm][l + 1] = g[(unsigned)((s * t.Nm + mc) * t.Nl + min(l, t.Nl - 1)) * pl + zk];
    }
    float2 graw[MAXL];                                     // G_{l,m} (hyper-viscosity acts on G, not H)
#pragma unroll
    for (int l = 0; l < MAXL; ++l) graw[l] = h[2][l + 1];
#pragma unroll
    for (int dm = 0; dm < 5; ++dm) {
        const int mm = m + dm - 2;
        const bool mv = mm >= 0 && mm < t.Nm;
#pragma unroll
        for (int l = 0; l < MAXL; ++l) {
            float2 v = h[dm][l + 1];
            if (!(mv && l < t.Nl)) v = make_float2(0.f, 0.f);
            else if (mm == 0) { v.x = fmaf(zt * J[l + 1], f.x, v.x); v.y = fmaf(zt * J[l + 1], f.y, v.y); }
            h[dm][l + 1] = v;
        }
    }
    const float fm = (float)m;
    const float sm1 = sqrtf(fm + 1.f), sm0 = sqrtf(fm);
    const float cA = sqrtf((fm + 1.f) * (fm + 2.f)), cB = 2.f * fm + 1.f, cC = sqrtf(fm * fmaxf(fm - 1.f, 0.f));
    const float bg = -vt * t.bgrad[z];
    const float wk = tz * t.omd[zk], wb = tz * t.omd[pl + zk];
    const float hv = t.hypv[zk];
    const float dd = t.dend ? t.dend[zk] : 0.f;
    const float ky = t.dky * (float)(k % t.naky);
    const float b = t.bs[(unsigned)s * pl + zk];
    const float sb = sqrtf(fmaxf(b, 0.f));
    float2 up = make_float2(0.f, 0.f), uq = up, tb = up;
    if (nu != 0.f && m <= 2) {
        const float2* __restrict__ mo = t.mom + (size_t)s * 3 * pl + zk;
        up = mo[0]; uq = mo[pl]; tb = mo[2 * (size_t)pl];
    }
#pragma unroll
    for (int l = 0; l < MAXL; ++l) {
        if (l < t.Nl) {
            const float fl = (float)l;
            const float2 c0 = h[2][l + 1];
            // mirror force
            const float ca = -(fl + 1.f) * sm1, cb = -fl * sm1, cc = fl * sm0, cd = (fl + 1.f) * sm0;
            float2 r;
            r.x = bg * (ca * h[3][l + 1].x + cb * h[3][l].x + cc * h[1][l + 1].x + cd * h[1][l + 2].x);
            r.y = bg * (ca * h[3][l + 1].y + cb * h[3][l].y + cc * h[1][l + 1].y + cd * h[1][l + 2].y);
            // drifts: -i (tau/Z) w (...)
            const float bx = wk * (cA * h[4][l + 1].x + cB * c0.x + cC * h[0][l + 1].x) +
                             wb * ((fl + 1.f) * h[2][l + 2].x + (2.f * fl + 1.f) * c0.x + fl * h[2][l].x);
            const float by = wk * (cA * h[4][l + 1].y + cB * c0.y + cC * h[0][l + 1].y) +
                             wb * ((fl + 1.f) * h[2][l + 2].y + (2.f * fl + 1.f) * c0.y + fl * h[2][l].y);
            r.x += by;
            r.y -= bx;
            const float jm = J[l], j0 = J[l + 1], jp = J[l + 2];
            const float jt = fl * jm + 2.f * fl * j0 + (fl + 1.f) * jp;
            if (m == 0 || m == 2) {                          // drive
                const float c = m == 0 ? t.fprim[s] * j0 + t.tprim[s] * jt : t.tprim[s] * j0 * 0.70710678118654752440f;
                r.x -= ky * c * f.y;
                r.y += ky * c * f.x;
            }
            if (nu != 0.f) {                                 // Dougherty
                const float damp = nu * (b + 2.f * fl + fm);
                r.x -= damp * c0.x;
                r.y -= damp * c0.y;
                if (m == 0) {
                    const float cu = sb * (j0 + jm), ct = 2.f * jt;
                    r.x = fmaf(nu, cu * uq.x + ct * tb.x, r.x);
                    r.y = fmaf(nu, cu * uq.y + ct * tb.y, r.y);
                } else if (m == 1) {
                    r.x = fmaf(nu * j0, up.x, r.x);
                    r.y = fmaf(nu * j0, up.y, r.y);
                } else if (m == 2) {
                    r.x = fmaf(nu * 1.41421356237309504880f * j0, tb.x, r.x);
                    r.y = fmaf(nu * 1.41421356237309504880f * j0, tb.y, r.y);
                }
            }
            // hyper-viscosity
            r.x -= hv * graw[l].x;
            r.y -= hv * graw[l].y;
            // wave-absorbing end layer (Eq. 4.30)
            r.x -= dd * c0.x;
            r.y -= dd * c0.y;
            float2* __restrict__ o = out + ((unsigned)((s * t.Nm + m) * t.Nl + l) * pl + zk);
            if (ACC) { const float2 prev = *o; r.x += prev.x; r.y += prev.y; }
            *o = r;
        }
    }
}

// The same pointwise terms, marching along the Hermite index: one thread per (s, z, k) walks m = m0 .. m1-1 with the
// five stencil planes H_{.,m-2..m+2} (all l) in registers, loads every G value exactly once (plane m+3 is requested
// while m is evaluated) and reads the (s,z,k) tables once.  lin_point_kernel relies on L2 for the five-fold reuse
// in m and keeps one batch of loads per thread in flight: ncu showed it latency-bound at 18 % of the DRAM bandwidth
// (long scoreboard 7.7 per issue, 15 warps per SM; profiles/r02_linear.md).  gridDim.z splits the m range when
// Ns*Nz*nk alone does not fill the machine (each chunk re-reads its four halo planes).
template <int MAXL, bool ACC>
__global__ void __launch_bounds__(128) lin_point_march_kernel(LinTables t, const float2* __restrict__ g,
                                                              const float2* __restrict__ phi, float2* __restrict__ out,
                                                              const int mchunk) {
    const unsigned pl = (unsigned)(t.Nz * t.nk);
    const unsigned zk = blockIdx.x * blockDim.x + threadIdx.x;
    if (zk >= pl) return;
    const int s = blockIdx.y;
    const int m0 = blockIdx.z * mchunk, m1 = min(t.Nm, m0 + mchunk);
    const int z = zk / t.nk, k = zk - z * t.nk;
    const float zt = t.zt[s], vt = t.vt[s], tz = t.tz[s], nu = t.nu[s];
    const float2 f = phi[zk];
    float J[MAXL + 2];                                     // J[l + 1] = J_l, zero outside 0 <= l < Nl
    J[0] = 0.f;
#pragma unroll
    for (int l = 0; l < MAXL; ++l) J[l + 1] = l < t.Nl ? t.Jl[(unsigned)(s * t.Nl + l) * pl + zk] : 0.f;
    J[MAXL + 1] = 0.f;
    const float bg = -vt * t.bgrad[z];
    const float wk = tz * t.omd[zk], wb = tz * t.omd[pl + zk];
    const float hv = t.hypv[zk];
    const float dd = t.dend ? t.dend[zk] : 0.f;
    const float ky = t.dky * (float)(k % t.naky);
    const float b = t.bs[(unsigned)s * pl + zk];
    const float sb = sqrtf(fmaxf(b, 0.f));
    float2 up = make_float2(0.f, 0.f), uq = up, tb = up;
    if (nu != 0.f && m0 <= 2) {
        const float2* __restrict__ mo = t.mom + (size_t)s * 3 * pl + zk;
        up = mo[0]; uq = mo[pl]; tb = mo[2 * (size_t)pl];
    }
    // H_{l,mm} = G_{l,mm} + (Z/tau) J_l Phi delta_{mm,0}; zero outside 0 <= mm < Nm, 0 <= l < Nl
    auto load_plane = [&](const int mm, float2 (&row)[MAXL + 2]) {
        row[0] = row[MAXL + 1] = make_float2(0.f, 0.f);
        const bool mv = mm >= 0 && mm < t.Nm;
        const int mc = min(max(mm, 0), t.Nm - 1);
#pragma unroll
        for (int l = 0; l < MAXL; ++l) {
            float2 v = g[(unsigned)((s * t.Nm + mc) * t.Nl + min(l, t.Nl - 1)) * pl + zk];     // unconditional: all in flight
            if (!(mv && l < t.Nl)) v = make_float2(0.f, 0.f);
            else if (mm == 0) { v.x = fmaf(zt * J[l + 1], f.x, v.x); v.y = fmaf(zt * J[l + 1], f.y, v.y); }
            row[l + 1] = v;
        }
    };
    float2 h[6][MAXL + 2];                                 // h[i] = plane m - 2 + i; h[5] is the plane in flight
#pragma unroll
    for (int i = 0; i < 5; ++i) load_plane(m0 - 2 + i, h[i]);
    for (int m = m0; m < m1; ++m) {
        load_plane(m + 3, h[5]);
        const float fm = (float)m;
        const float sm1 = sqrtf(fm + 1.f), sm0 = sqrtf(fm);
        const float cA = sqrtf((fm + 1.f) * (fm + 2.f)), cB = 2.f * fm + 1.f, cC = sqrtf(fm * fmaxf(fm - 1.f, 0.f));
#pragma unroll
        for (int l = 0; l < MAXL; ++l) {
            if (l < t.Nl) {
                const float fl = (float)l;
                const float2 c0 = h[2][l + 1];
                // mirror force
                const float ca = -(fl + 1.f) * sm1, cb = -fl * sm1, cc = fl * sm0, cd = (fl + 1.f) * sm0;
                float2 r;
                r.x = bg * (ca * h[3][l + 1].x + cb * h[3][l].x + cc * h[1][l + 1].x + cd * h[1][l + 2].x);
                r.y = bg * (ca * h[3][l + 1].y + cb * h[3][l].y + cc * h[1][l + 1].y + cd * h[1][l + 2].y);
                // drifts: -i (tau/Z) w (...)
                const float bx = wk * (cA * h[4][l + 1].x + cB * c0.x + cC * h[0][l + 1].x) +
                                 wb * ((fl + 1.f) * h[2][l + 2].x + (2.f * fl + 1.f) * c0.x + fl * h[2][l].x);
                const float by = wk * (cA * h[4][l + 1].y + cB * c0.y + cC * h[0][l + 1].y) +
                                 wb * ((fl + 1.f) * h[2][l + 2].y + (2.f * fl + 1.f) * c0.y + fl * h[2][l].y);
                r.x += by;
                r.y -= bx;
                const float jm = J[l], j0 = J[l + 1], jp = J[l + 2];
                const float jt = fl * jm + 2.f * fl * j0 + (fl + 1.f) * jp;
                if (m == 0 || m == 2) {                          // drive
                    const float c = m == 0 ? t.fprim[s] * j0 + t.tprim[s] * jt : t.tprim[s] * j0 * 0.70710678118654752440f;
                    r.x -= ky * c * f.y;
                    r.y += ky * c * f.x;
                }
                if (nu != 0.f) {                                 // Dougherty
                    const float damp = nu * (b + 2.f * fl + fm);
                    r.x -= damp * c0.x;
                    r.y -= damp * c0.y;
                    if (m == 0) {
                        const float cu = sb * (j0 + jm), ct = 2.f * jt;
                        r.x = fmaf(nu, cu * uq.x + ct * tb.x, r.x);
                        r.y = fmaf(nu, cu * uq.y + ct * tb.y, r.y);
                    } else if (m == 1) {
                        r.x = fmaf(nu * j0, up.x, r.x);
                        r.y = fmaf(nu * j0, up.y, r.y);
                    } else if (m == 2) {
                        r.x = fmaf(nu * 1.41421356237309504880f * j0, tb.x, r.x);
                        r.y = fmaf(nu * 1.41421356237309504880f * j0, tb.y, r.y);
                    }
                }
                // hyper-viscosity acts on G, not H
                const float gx_ = m == 0 ? c0.x - zt * j0 * f.x : c0.x, gy_ = m == 0 ? c0.y - zt * j0 * f.y : c0.y;
                r.x -= hv * gx_;
                r.y -= hv * gy_;
                // wave-absorbing end layer (Eq. 4.30)
                r.x -= dd * c0.x;
                r.y -= dd * c0.y;
                float2* __restrict__ o = out + ((unsigned)((s * t.Nm + m) * t.Nl + l) * pl + zk);
                if (ACC) { const float2 prev = *o; r.x += prev.x; r.y += prev.y; }
                *o = r;
            }
        }
#pragma unroll
        for (int i = 0; i < 5; ++i)
#pragma unroll
            for (int l = 0; l < MAXL + 2; ++l) h[i][l] = h[i + 1][l];
    }
}

// Twist-and-shift linked z operators (Eq. 4.29): one block per (slice of a chain of linked modes,
// l, (s,m)); the chain's extended periodic domain (L segments of Nz points, in order of increasing ballooning
// angle) is staged in shared memory and the two circulant products of the slice's outputs are added to out.
template <int ZB>
__global__ void __launch_bounds__(kZlinkThreads) lin_zlink_kernel(LinTables t, const float2* __restrict__ g,
                                                                  const float2* __restrict__ phi,
                                                                  float2* __restrict__ out, const int work0,
                                                                  const int cap) {
    extern __shared__ __align__(16) unsigned char lin_smem[];
    const int c = t.zwork[work0 + blockIdx.x] >> 8, slice = t.zwork[work0 + blockIdx.x] & 255;
    const int s = blockIdx.z / t.Nm, m = blockIdx.z % t.Nm;
    const int off = t.chain_off[c], L = t.chain_off[c + 1] - off, N = L * t.Nz;
    float2* S1 = reinterpret_cast<float2*>(lin_smem);            // [N]
    float2* S2 = S1 + cap;                                       // [N]   (cap >= N: points the launch provides for)
    float* dcol = reinterpret_cast<float*>(S2 + cap);            // [2N] column repeated
    float* acol = dcol + 2 * cap;
    int* modes = reinterpret_cast<int*>(acol + 2 * cap);         // [L]
    const float* __restrict__ ed = t.ext_d + t.ext_off[c];
    const float* __restrict__ ea = t.ext_a + t.ext_off[c];
    const float hyp = t.nuhyp[s] * t.mpow[m], vt = t.vt[s];
    for (int i = threadIdx.x; i < 2 * N; i += blockDim.x) {
        const int d = i < N ? i : i - N;
        dcol[i] = ed[d];
        acol[i] = ea[d];
    }
    for (int i = threadIdx.x; i < L; i += blockDim.x) modes[i] = t.chain_mode[off + i];
    const unsigned pl = (unsigned)(t.Nz * t.nk);
    const bool vp = m + 1 < t.Nm, vm = m - 1 >= 0;
    const float cp = vp ? sqrtf((float)(m + 1)) : 0.f, cm = vm ? sqrtf((float)m) : 0.f;
    const float cphi = (vm && m == 1) ? cm * t.zt[s] : 0.f;
    {
        const int l = blockIdx.y;
        __syncthreads();
        const unsigned ip = (unsigned)((s * t.Nm + (vp ? m + 1 : m)) * t.Nl + l) * pl,
                       im = (unsigned)((s * t.Nm + (vm ? m - 1 : m)) * t.Nl + l) * pl,
                       i0 = (unsigned)((s * t.Nm + m) * t.Nl + l) * pl, ij = (unsigned)(s * t.Nl + l) * pl;
        for (int i = threadIdx.x; i < N; i += blockDim.x) {
            const int seg = i / t.Nz, z = i - seg * t.Nz;
            const unsigned zk = (unsigned)(z * t.nk + modes[seg]);
            const float2 a = g[ip + zk], b = g[im + zk];
            float2 v = make_float2(cp * a.x + cm * b.x, cp * a.y + cm * b.y);
            if (cphi != 0.f) {
                const float w = cphi * t.Jl[ij + zk];
                const float2 f = phi[zk];
                v.x = fmaf(w, f.x, v.x);
                v.y = fmaf(w, f.y, v.y);
            }
            S1[i] = v;
            S2[i] = g[i0 + zk];
        }
        __syncthreads();
        const int lo = slice * kZlinkSlice, hi = min(N, lo + kZlinkSlice);
        for (int z0 = lo + threadIdx.x * ZB; z0 < hi; z0 += blockDim.x * ZB) {
            float2 dp[ZB], ap[ZB];
#pragma unroll
            for (int i = 0; i < ZB; ++i) dp[i] = ap[i] = make_float2(0.f, 0.f);
            auto blocked = [&](const float* __restrict__ col, const float2* __restrict__ sv, float2 (&acc)[ZB]) {
                const float* __restrict__ dc = col + z0 + N;               // weight of (z0 + i, zp) = dc[i - zp]
                if constexpr (ZB == 4) {
                    float w0 = dc[0], w1 = dc[1], w2 = dc[2], w3 = dc[3];
                    for (int zp = 0; zp < N; zp += 4) {
                        const float2 a0 = sv[zp], a1 = sv[zp + 1], a2 = sv[zp + 2], a3 = sv[zp + 3];
                        const float n0 = dc[-(zp + 1)], n1 = dc[-(zp + 2)], n2 = dc[-(zp + 3)], n3 = dc[-(zp + 4)];
                        acc[0].x = fmaf(w0, a0.x, acc[0].x); acc[0].y = fmaf(w0, a0.y, acc[0].y);
                        acc[1].x = fmaf(w1, a0.x, acc[1].x); acc[1].y = fmaf(w1, a0.y, acc[1].y);
                        acc[2].x = fmaf(w2, a0.x, acc[2].x); acc[2].y = fmaf(w2, a0.y, acc[2].y);
                        acc[3].x = fmaf(w3, a0.x, acc[3].x); acc[3].y = fmaf(w3, a0.y, acc[3].y);
                        acc[0].x = fmaf(n0, a1.x, acc[0].x); acc[0].y = fmaf(n0, a1.y, acc[0].y);
                        acc[1].x = fmaf(w0, a1.x, acc[1].x); acc[1].y = fmaf(w0, a1.y, acc[1].y);
                        acc[2].x = fmaf(w1, a1.x, acc[2].x); acc[2].y = fmaf(w1, a1.y, acc[2].y);
                        acc[3].x = fmaf(w2, a1.x, acc[3].x); acc[3].y = fmaf(w2, a1.y, acc[3].y);
                        acc[0].x = fmaf(n1, a2.x, acc[0].x); acc[0].y = fmaf(n1, a2.y, acc[0].y);
                        acc[1].x = fmaf(n0, a2.x, acc[1].x); acc[1].y = fmaf(n0, a2.y, acc[1].y);
                        acc[2].x = fmaf(w0, a2.x, acc[2].x); acc[2].y = fmaf(w0, a2.y, acc[2].y);
                        acc[3].x = fmaf(w1, a2.x, acc[3].x); acc[3].y = fmaf(w1, a2.y, acc[3].y);
                        acc[0].x = fmaf(n2, a3.x, acc[0].x); acc[0].y = fmaf(n2, a3.y, acc[0].y);
                        acc[1].x = fmaf(n1, a3.x, acc[1].x); acc[1].y = fmaf(n1, a3.y, acc[1].y);
                        acc[2].x = fmaf(n0, a3.x, acc[2].x); acc[2].y = fmaf(n0, a3.y, acc[2].y);
                        acc[3].x = fmaf(w0, a3.x, acc[3].x); acc[3].y = fmaf(w0, a3.y, acc[3].y);
                        w3 = n0; w2 = n1; w1 = n2; w0 = n3;
                    }
                } else {
                    for (int zp = 0; zp < N; ++zp) {
                        const float w = dc[-zp];
                        acc[0].x = fmaf(w, sv[zp].x, acc[0].x); acc[0].y = fmaf(w, sv[zp].y, acc[0].y);
                    }
                }
            };
            blocked(dcol, S1, dp);
            if (hyp != 0.f) blocked(acol, S2, ap);
#pragma unroll
            for (int i = 0; i < ZB; ++i) {
                const int zi = z0 + i, seg = zi / t.Nz, z = zi - seg * t.Nz;
                float2* __restrict__ o = out + (i0 + (unsigned)(z * t.nk + modes[seg]));
                const float2 prev = *o;
                *o = make_float2(prev.x - vt * dp[i].x - hyp * ap[i].x, prev.y - vt * dp[i].y - hyp * ap[i].y);
            }
        }
    }
}

// The same two operators for the LONG chains, in the harmonics of the extended domain.  N = L*Nz factorises: with point
// n = Nz*n1 + n2 (segment n1, point n2) and harmonic jj = k1 + L*k2,
//   X[k1 + L k2] = sum_n2 W_Nz^{n2 k2} W_N^{n2 k1} sum_n1 W_L^{n1 k1} x[Nz n1 + n2],        W_M = e^{-2 pi i/M},
// i.e. a dense DFT over the L segments for every point of a segment, a twiddle and a dense Nz-point DFT per k1:
// N (L + Nz) multiply-adds per transform instead of the N^2 of the circulant product (N up to 26 x 24 = 624 on the Cyclone
// grid).  The operators are diagonal there, grad_par -> i gradpar j/L and |k_par| -> |gradpar| |j|/L for the signed
// harmonic j (Nyquist dropped for the derivative, as in the table build above); one inverse transform of their sum.
// One block per (chain, l, (s,m)); shared memory: X1, X2, T1, T2, W_N tables of N complex, W_L, W_Nz, the chain's modes.
constexpr int kZspecThreads = 128;
__global__ void __launch_bounds__(kZspecThreads) lin_zlink_spectral_kernel(LinTables t, const float2* __restrict__ g,
                                                                          const float2* __restrict__ phi,
                                                                          float2* __restrict__ out, const int cap) {
    extern __shared__ __align__(16) unsigned char lin_smem[];
    const int c = t.zlong[blockIdx.x];
    const int s = blockIdx.z / t.Nm, m = blockIdx.z % t.Nm, l = blockIdx.y;
    const int off = t.chain_off[c], L = t.chain_off[c + 1] - off, Nz = t.Nz, N = L * Nz;
    float2* X1 = reinterpret_cast<float2*>(lin_smem);      // sqrt(m+1) H_{l,m+1} + sqrt(m) H_{l,m-1}; later the spectrum of the sum
    float2* X2 = X1 + cap;                                  // G_{l,m}
    float2* T1 = X2 + cap;
    float2* T2 = T1 + cap;
    float2* WN = T2 + cap;                                  // e^{-2 pi i j/N}
    float2* WL = WN + cap;                                  // e^{-2 pi i j/L}, L <= cap/Nz
    float2* WZ = WL + cap / Nz;                             // e^{-2 pi i j/Nz}
    int* modes = reinterpret_cast<int*>(WZ + Nz);
    const int tid = threadIdx.x;
    for (int i = tid; i < N; i += kZspecThreads) { float sn, cs; sincospif(-2.f * (float)i / (float)N, &sn, &cs); WN[i] = make_float2(cs, sn); }
    for (int i = tid; i < L; i += kZspecThreads) { float sn, cs; sincospif(-2.f * (float)i / (float)L, &sn, &cs); WL[i] = make_float2(cs, sn); modes[i] = t.chain_mode[off + i]; }
    for (int i = tid; i < Nz; i += kZspecThreads) { float sn, cs; sincospif(-2.f * (float)i / (float)Nz, &sn, &cs); WZ[i] = make_float2(cs, sn); }
    const unsigned pl = (unsigned)(Nz * t.nk);
    const bool vp = m + 1 < t.Nm, vm = m - 1 >= 0;
    const float cp = vp ? sqrtf((float)(m + 1)) : 0.f, cm = vm ? sqrtf((float)m) : 0.f;
    const float cphi = (vm && m == 1) ? cm * t.zt[s] : 0.f;
    const float hyp = t.nuhyp[s] * t.mpow[m], vt = t.vt[s];
    const unsigned ip = (unsigned)((s * t.Nm + (vp ? m + 1 : m)) * t.Nl + l) * pl,
                   im = (unsigned)((s * t.Nm + (vm ? m - 1 : m)) * t.Nl + l) * pl,
                   i0 = (unsigned)((s * t.Nm + m) * t.Nl + l) * pl, ij = (unsigned)(s * t.Nl + l) * pl;
    __syncthreads();
    for (int i = tid; i < N; i += kZspecThreads) {
        const int seg = i / Nz, z = i - seg * Nz;
        const unsigned zk = (unsigned)(z * t.nk + modes[seg]);
        const float2 a = g[ip + zk], b = g[im + zk];
        float2 v = make_float2(cp * a.x + cm * b.x, cp * a.y + cm * b.y);
        if (cphi != 0.f) {
            const float w = cphi * t.Jl[ij + zk];
            const float2 f = phi[zk];
            v.x = fmaf(w, f.x, v.x);
            v.y = fmaf(w, f.y, v.y);
        }
        X1[i] = v;
        X2[i] = g[i0 + zk];
    }
    __syncthreads();
    const bool with_hyp = hyp != 0.f;
    // ---- forward, step A: T[k1*Nz + n2] = W_N^{n2 k1} sum_n1 W_L^{n1 k1} x[Nz n1 + n2]
    for (int i = tid; i < N; i += kZspecThreads) {
        const int k1 = i / Nz, n2 = i - k1 * Nz;
        float2 a1 = make_float2(0.f, 0.f), a2 = a1;
        int w = 0;                                          // (n1 k1) mod L
        for (int n1 = 0; n1 < L; ++n1) {
            const float2 tw = WL[w];
            const float2 x1 = X1[n1 * Nz + n2];
            a1.x = fmaf(tw.x, x1.x, fmaf(-tw.y, x1.y, a1.x)); a1.y = fmaf(tw.x, x1.y, fmaf(tw.y, x1.x, a1.y));
            if (with_hyp) {
                const float2 x2 = X2[n1 * Nz + n2];
                a2.x = fmaf(tw.x, x2.x, fmaf(-tw.y, x2.y, a2.x)); a2.y = fmaf(tw.x, x2.y, fmaf(tw.y, x2.x, a2.y));
            }
            w += k1; if (w >= L) w -= L;
        }
        const float2 tn = WN[(n2 * k1) % N];
        T1[i] = make_float2(a1.x * tn.x - a1.y * tn.y, a1.x * tn.y + a1.y * tn.x);
        T2[i] = make_float2(a2.x * tn.x - a2.y * tn.y, a2.x * tn.y + a2.y * tn.x);
    }
    __syncthreads();
    // ---- forward, step B: X[k1 + L k2] = sum_n2 W_Nz^{n2 k2} T[k1*Nz + n2]; the operators; the sum's spectrum -> X1[k1*Nz + k2]
    const float cd = -vt * t.gradpar / (float)L, ca = -hyp * fabsf(t.gradpar) / (float)L;
    for (int i = tid; i < N; i += kZspecThreads) {
        const int k1 = i / Nz, kk2 = i - k1 * Nz;
        float2 b1 = make_float2(0.f, 0.f), b2 = b1;
        int w = 0;                                          // (n2 k2) mod Nz
        for (int n2 = 0; n2 < Nz; ++n2) {
            const float2 tw = WZ[w];
            const float2 x1 = T1[k1 * Nz + n2];
            b1.x = fmaf(tw.x, x1.x, fmaf(-tw.y, x1.y, b1.x)); b1.y = fmaf(tw.x, x1.y, fmaf(tw.y, x1.x, b1.y));
            if (with_hyp) {
                const float2 x2 = T2[k1 * Nz + n2];
                b2.x = fmaf(tw.x, x2.x, fmaf(-tw.y, x2.y, b2.x)); b2.y = fmaf(tw.x, x2.y, fmaf(tw.y, x2.x, b2.y));
            }
            w += kk2; if (w >= Nz) w -= Nz;
        }
        const int jj = k1 + L * kk2;
        const int j = jj <= N / 2 ? jj : jj - N;
        const float fd = (N % 2 == 0 && jj == N / 2) ? 0.f : cd * (float)j;      // -v_t * (i gradpar j/L): times i below
        const float fa = ca * fabsf((float)j);
        X1[i] = make_float2(-fd * b1.y + fa * b2.x, fd * b1.x + fa * b2.y);
    }
    __syncthreads();
    // ---- inverse, step C: U[k1*Nz + n2] = conj W_N^{n2 k1} sum_k2 conj W_Nz^{n2 k2} Y[k1 + L k2]
    for (int i = tid; i < N; i += kZspecThreads) {
        const int k1 = i / Nz, n2 = i - k1 * Nz;
        float2 u = make_float2(0.f, 0.f);
        int w = 0;
        for (int kk2 = 0; kk2 < Nz; ++kk2) {
            const float2 tw = WZ[w];
            const float2 y = X1[k1 * Nz + kk2];
            u.x = fmaf(tw.x, y.x, fmaf(tw.y, y.y, u.x)); u.y = fmaf(tw.x, y.y, fmaf(-tw.y, y.x, u.y));      // y * conj(tw)
            w += n2; if (w >= Nz) w -= Nz;
        }
        const float2 tn = WN[(n2 * k1) % N];
        T1[i] = make_float2(u.x * tn.x + u.y * tn.y, u.y * tn.x - u.x * tn.y);
    }
    __syncthreads();
    // ---- inverse, step D: y[Nz n1 + n2] = (1/N) sum_k1 conj W_L^{n1 k1} U[k1*Nz + n2]; added to out
    const float rn = 1.f / (float)N;
    for (int i = tid; i < N; i += kZspecThreads) {
        const int n1 = i / Nz, n2 = i - n1 * Nz;
        float2* __restrict__ o = out + (i0 + (unsigned)(n2 * t.nk + modes[n1]));
        const float2 prev = *o;                             // requested before the sum
        float2 y = make_float2(0.f, 0.f);
        int w = 0;
        for (int k1 = 0; k1 < L; ++k1) {
            const float2 tw = WL[w];
            const float2 u = T1[k1 * Nz + n2];
            y.x = fmaf(tw.x, u.x, fmaf(tw.y, u.y, y.x)); y.y = fmaf(tw.x, u.y, fmaf(-tw.y, u.x, y.y));
            w += n1; if (w >= L) w -= L;
        }
        *o = make_float2(fmaf(rn, y.x, prev.x), fmaf(rn, y.y, prev.y));
    }
}

// Launches the pointwise terms: the marching kernel (one thread per (s,z,k), m range split over gridDim.z until about
// 130 k threads exist) unless GX_LIN_POINT=stencil asks for the per-(s,m) stencil kernel.
template <int MAXL>
inline void launch_lin_point(const LinTables& t, const float2* g, const float2* phi, float2* out, bool accumulate, cudaStream_t st) {
    const char* lp = std::getenv("GX_LIN_POINT");            // read per call: the tests switch it
    const bool stencil = lp && std::strcmp(lp, "stencil") == 0;
    const size_t pl = (size_t)t.Nz * t.nk;
    if (stencil) {
        dim3 gp(t.Ns * t.Nm, (unsigned)((pl + 255) / 256));
        if (accumulate) lin_point_kernel<MAXL, true><<<gp, 256, 0, st>>>(t, g, phi, out);
        else lin_point_kernel<MAXL, false><<<gp, 256, 0, st>>>(t, g, phi, out);
        return;
    }
    int chunks = (int)((130000 + (size_t)t.Ns * pl - 1) / ((size_t)t.Ns * pl));     // measured: 2 chunks for Cyclone and kinetic, 1 above
    static const int forced = std::getenv("GX_LIN_CHUNKS") ? std::atoi(std::getenv("GX_LIN_CHUNKS")) : 0;     // tuning aid
    if (forced > 0) chunks = forced;
    chunks = std::max(1, std::min(chunks, std::max(1, t.Nm / (forced > 0 ? 1 : 2))));
    const int mchunk = (t.Nm + chunks - 1) / chunks;
    dim3 gp((unsigned)((pl + 127) / 128), t.Ns, (t.Nm + mchunk - 1) / mchunk);      // 128 threads: 117-183 registers each
    if (accumulate) lin_point_march_kernel<MAXL, true><<<gp, 128, 0, st>>>(t, g, phi, out, mchunk);
    else lin_point_march_kernel<MAXL, false><<<gp, 128, 0, st>>>(t, g, phi, out, mchunk);
}

// Opt-in shared-memory sizes of every linear kernel instantiation, on the current device (gx_grid_create: per
// handle and per device, no process-wide cache).
inline cudaError_t lin_prepare() {
    constexpr int kMax = 200 * 1024;
    cudaError_t e = cudaSuccess;
#define GX_ATTR(K) if (e == cudaSuccess) e = cudaFuncSetAttribute(K, cudaFuncAttributeMaxDynamicSharedMemorySize, kMax)
    GX_ATTR((lin_rhs_kernel<true, 4>));  GX_ATTR((lin_rhs_kernel<false, 4>));
    GX_ATTR((lin_rhs_kernel<true, 1>));  GX_ATTR((lin_rhs_kernel<false, 1>));
    GX_ATTR((lin_rhs_kernel<true, 4, true>));  GX_ATTR((lin_rhs_kernel<true, 1, true>));
    GX_ATTR((lin_rhs_kernel<true, 1, true, 8, 8>));   GX_ATTR((lin_rhs_kernel<true, 1, false, 8, 8>));   GX_ATTR((lin_rhs_kernel<false, 1, false, 8, 8>));
    GX_ATTR((lin_rhs_kernel<true, 1, true, 8, 12>));  GX_ATTR((lin_rhs_kernel<true, 1, false, 8, 12>));  GX_ATTR((lin_rhs_kernel<false, 1, false, 8, 12>));
    GX_ATTR((lin_rhs_kernel<true, 1, true, 8, 16>));  GX_ATTR((lin_rhs_kernel<true, 1, false, 8, 16>));  GX_ATTR((lin_rhs_kernel<false, 1, false, 8, 16>));
    GX_ATTR(lin_zlink_kernel<4>);  GX_ATTR(lin_zlink_kernel<1>);  GX_ATTR(lin_zlink_spectral_kernel);
#undef GX_ATTR
    return e;
}

inline cudaError_t lin_rhs(const LinTables& t, const float2* g, const float2* phi, float2* out, bool accumulate,
                           cudaStream_t st) {
    if (!t.built) return cudaErrorNotReady;
    if (t.any_nu) {
        dim3 gm((t.nk + 255) / 256, t.Nz, t.Ns);
        lin_moments_kernel<<<gm, 256, 0, st>>>(t, g, phi);
    }
    const int fa = (t.Nz == 64 || t.Nz == 96 || t.Nz == 128) ? 8 : 0;      // z FFT path: Nz = 8 x {8, 12, 16}
    const size_t smem = (size_t)t.Nz * kLinTK * sizeof(float2) * (fa ? 3 : 2) + 4 * (size_t)t.Nz * sizeof(float);
    if (fa && !t.linked) {
        cudaError_t e = cudaSuccess;
        dim3 gridf(t.Ns * t.Nm, t.Nl, (t.nk + kLinTK - 1) / kLinTK);
        const bool splitf = t.Nl <= 6;        // pointwise terms with the stencil in registers, z operators added on top
        if (splitf) {
            if (t.Nl <= 4) {
                launch_lin_point<4>(t, g, phi, out, accumulate, st);
            } else {
                launch_lin_point<6>(t, g, phi, out, accumulate, st);
            }
        }
#define GX_ZFFT(FB)                                                                                                        \
    do {                                                                                                                   \
        if (splitf) {                                                                                                      \
            lin_rhs_kernel<true, 1, true, 8, FB><<<gridf, kLinTK * kLinZG, smem, st>>>(t, g, phi, out, false);  \
        } else if (accumulate) {                                                                                           \
            lin_rhs_kernel<true, 1, false, 8, FB><<<gridf, kLinTK * kLinZG, smem, st>>>(t, g, phi, out, false); \
        } else {                                                                                                           \
            lin_rhs_kernel<false, 1, false, 8, FB><<<gridf, kLinTK * kLinZG, smem, st>>>(t, g, phi, out, false); \
        }                                                                                                                  \
    } while (0)
        if (t.Nz == 64) GX_ZFFT(8);
        else if (t.Nz == 96) GX_ZFFT(12);
        else GX_ZFFT(16);
#undef GX_ZFFT
        return e != cudaSuccess ? e : cudaGetLastError();
    }
    dim3 grid(t.Ns * t.Nm, t.Nl, (t.nk + kLinTK - 1) / kLinTK);
    const bool b4 = t.Nz % 4 == 0;
    static const bool fused8 = std::getenv("GX_LIN_FUSED8") != nullptr;      // development aid: the round-1 choice for Nl > 4
    const bool split = t.Nl <= 4 || t.linked || !fused8;
    if (split && t.Nl <= 8) {
        // pointwise terms (marching kernel), then the z-operator terms added on top.  With the per-(s,m) stencil kernel
        // this paid for Nl <= 4 only (5 x 10 stencil values, 135 registers); with the marching kernel it pays for Nl = 8 too
        if (t.Nl <= 4) {
            launch_lin_point<4>(t, g, phi, out, accumulate, st);
        } else {
            launch_lin_point<8>(t, g, phi, out, accumulate, st);
        }
        if (!t.linked) {
            if (b4) lin_rhs_kernel<true, 4, true><<<grid, kLinTK * kLinZG, smem, st>>>(t, g, phi, out, false);
            else lin_rhs_kernel<true, 1, true><<<grid, kLinTK * kLinZG, smem, st>>>(t, g, phi, out, false);
        }
    } else if (accumulate) {
        if (b4) lin_rhs_kernel<true, 4><<<grid, kLinTK * kLinZG, smem, st>>>(t, g, phi, out, t.linked);
        else lin_rhs_kernel<true, 1><<<grid, kLinTK * kLinZG, smem, st>>>(t, g, phi, out, t.linked);
    } else {
        if (b4) lin_rhs_kernel<false, 4><<<grid, kLinTK * kLinZG, smem, st>>>(t, g, phi, out, t.linked);
        else lin_rhs_kernel<false, 1><<<grid, kLinTK * kLinZG, smem, st>>>(t, g, phi, out, t.linked);
    }
    if (t.linked) {
        // two launches: the few long chains with room for the longest extended domain, the many short ones
        // (up to 4 links) with a small footprint so that 32 blocks fit an SM
        const int w0[2] = {0, t.nzwork_long}, wn[2] = {t.nzwork_long, t.nzwork - t.nzwork_long};
        const int cap[2] = {t.max_ext, t.short_ext};
        const char* zl = std::getenv("GX_ZLINK");               // "dense": the circulant products for the long chains too
        const bool spectral = t.nzlong > 0 && !(zl && std::strcmp(zl, "dense") == 0);
        if (spectral) {
            const size_t sm = (size_t)t.max_ext * 5 * sizeof(float2) + (size_t)(t.max_ext / t.Nz + t.Nz) * sizeof(float2) +
                              (size_t)(t.max_ext / t.Nz) * sizeof(int);
            if (sm > 200 * 1024) return cudaErrorInvalidConfiguration;
            dim3 gl(t.nzlong, t.Nl, t.Ns * t.Nm);
            lin_zlink_spectral_kernel<<<gl, kZspecThreads, sm, st>>>(t, g, phi, out, t.max_ext);
        }
        for (int part = spectral ? 1 : 0; part < 2; ++part) {
            if (wn[part] <= 0) continue;
            const size_t sm = (size_t)cap[part] * (2 * sizeof(float2) + 4 * sizeof(float)) + (size_t)(cap[part] / t.Nz) * sizeof(int);
            if (sm > 200 * 1024) return cudaErrorInvalidConfiguration;
            dim3 gl(wn[part], t.Nl, t.Ns * t.Nm);
            if (b4) lin_zlink_kernel<4><<<gl, kZlinkThreads, sm, st>>>(t, g, phi, out, w0[part], cap[part]);
            else lin_zlink_kernel<1><<<gl, kZlinkThreads, sm, st>>>(t, g, phi, out, w0[part], cap[part]);
        }
    }
    return cudaGetLastError();
}

// SSP-RK3 stage combine: out = a*y0 + b*(y + dt*k), element-wise; out may alias y0 or y.
__global__ void __launch_bounds__(256) rk_stage_kernel(float2* out, const float2* y0, const float2* y,
                                                       const float2* k, float a, float b, float dt, size_t n) {
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const float2 u = y0[i], v = y[i], w = k[i];
        out[i] = make_float2(fmaf(b, fmaf(dt, w.x, v.x), a * u.x), fmaf(b, fmaf(dt, w.y, v.y), a * u.y));
    }
}

}  // namespace gx
