// linear_kernels.cuh -- quasineutrality field solve and the linear terms of Eq. 4.9 (PAPER.md lines
// 212-260, 284, 298-318, 391) for gx_field_solve / gx_linear_rhs / gx_rhs.  SURVEY.md row f1.
//
// Tables are built on the host in fp64 and rounded once to fp32:
//   Jl[s][l][z][k]   = (1/l!)(-b_s/2)^l e^{-b_s/2}           Eq. 4.7 (line 202)
//   invD[z][k]       = 1 / ( sum_s Z^2 n/tau (1 - sum_l Jl^2) [+ Z^2 n/tau * tau_fac if adiabatic] )
//   fsfac[kx]        = pref*tau_fac / (1 - pref*tau_fac <<1/D>>)   (flux-surface-average closure, ky = 0)
#pragma once
#include <cuda_runtime.h>

#include <cmath>
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
    float* Dz = nullptr;       // [z][z'] gradpar * spectral d/dz
    float* Az = nullptr;       // [z][z'] gradpar * spectral |k_z|
    float* omd = nullptr;      // [2][z][k]  omega_d^kappa, omega_d^gradB
    float* hypv = nullptr;     // [z][k] D (kperp2/kperp2max)^n
    float* bgrad = nullptr;    // [z]
    float qn[kMaxSpecies] = {0}, zt[kMaxSpecies] = {0}, vt[kMaxSpecies] = {0}, tz[kMaxSpecies] = {0};
    float tprim[kMaxSpecies] = {0}, fprim[kMaxSpecies] = {0}, nu[kMaxSpecies] = {0}, nuhyp[kMaxSpecies] = {0};
    float dky = 0;
    bool built = false;
};

constexpr int kLinLaunchesFieldSolve = 2;
constexpr int kLinLaunchesRhs = 1;

inline void lin_tables_free(LinTables& t) {
    cudaFree(t.Jl); cudaFree(t.invD); cudaFree(t.fsfac); cudaFree(t.wz); cudaFree(t.bs);
    cudaFree(t.Dz); cudaFree(t.Az); cudaFree(t.omd); cudaFree(t.hypv); cudaFree(t.bgrad);
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
    (void)K;
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

// adiabatic electrons, ky = 0 rows: phi += fsfac[kx] * <<phi_raw>>_z * invD   (Eq. 6.1 solved for <<phi>>)
__global__ void __launch_bounds__(128) flux_surface_kernel(LinTables t, float2* __restrict__ phi) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;    // kx row
    if (i >= t.nakx || i == 0) return;
    const size_t col = (size_t)i * t.naky;
    float2 avg = make_float2(0.f, 0.f);
    for (int z = 0; z < t.Nz; ++z) {
        const float2 f = phi[(size_t)z * t.nk + col];
        avg.x = fmaf(t.wz[z], f.x, avg.x);
        avg.y = fmaf(t.wz[z], f.y, avg.y);
    }
    const float fs = t.fsfac[i];
    for (int z = 0; z < t.Nz; ++z) {
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
    if (t.adiabatic) flux_surface_kernel<<<(t.nakx + 127) / 128, 128, 0, st>>>(t, phi);
    return cudaGetLastError();
}

inline cudaError_t lin_rhs(const LinTables& t, const float2* g, const float2* phi, float2* out, bool accumulate,
                           cudaStream_t st) {
    (void)t; (void)g; (void)phi; (void)out; (void)accumulate; (void)st;
    return cudaErrorNotSupported;   // linear terms: next milestone
}

}  // namespace gx
