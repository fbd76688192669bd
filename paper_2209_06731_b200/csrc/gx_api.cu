// gx_api.cu -- host side of the C-ABI declared in include/gx.h: handle, tables (fp64 -> fp32 once),
// kernel dispatch.  No CPU compute path exists: every step of the hot path runs in nl_kernels.cuh.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstdint>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/gx.h"
#include "linear_kernels.cuh"
#include "kernel_sets.h"

namespace {

using gx::NlParams;

struct Species {
    double Z = 1, mass = 1, temp = 1, dens = 1, tprim = 0, fprim = 0, nu = 0;
    bool set = false;
};

using gxhost::KernelSet;
using gxhost::launch_pdl;

// Kernel families behind the one C-ABI ("Kernel families"; profiles/r02_rx_families.md):
//   row     (nl_row_kernels.cuh)   y direction of an x row in one thread's registers (NY = 64)   -- default where instantiated
//   scalar  (nl_kernels.cuh)       block-synchronous two-pass transforms, scalar FP32             -- default otherwise
//   rx      (nl_rx_kernels.cuh)    packed-FP32 x passes, packed C2R rows, a8 fused                -- GX_KERNELS=rx
//   rxp     (nl_rx_kernels.cuh)    rx phases in one persistent kernel, two groups per SM          -- GX_KERNELS=rxp
//   rxw     (nl_rx_kernels.cuh)    warp-specialised pipeline (row warps + x warps)                -- GX_KERNELS=rxw
// GX_KERNELS (read at gx_grid_create) forces a family; one without an instantiation for the grid falls through.
const KernelSet* find_set(int Nx, int Ny) {
    const char* fam = std::getenv("GX_KERNELS");
    const KernelSet* k = nullptr;
    if (fam && std::strcmp(fam, "rxw") == 0 && (k = gxhost::find_rx(Nx, Ny, GX_FAMILY_RXW))) return k;
    if (fam && std::strcmp(fam, "rxp") == 0 && (k = gxhost::find_rx(Nx, Ny, GX_FAMILY_RXP))) return k;
    if (fam && std::strcmp(fam, "rx") == 0 && (k = gxhost::find_rx(Nx, Ny, GX_FAMILY_RX))) return k;
    if ((!fam || std::strcmp(fam, "row") == 0) && (k = gxhost::find_row(Nx, Ny))) return k;
    return gxhost::find_scalar(Nx, Ny);
}

// ---------------------------------------------------------------------------- Gauss-Laguerre
// L_n(x) by the three-term recurrence (Eq. 4.3).
double laguerre(int n, double x) {
    double lm = 0.0, l = 1.0;
    for (int k = 0; k < n; ++k) {
        const double ln = ((2 * k + 1 - x) * l - k * lm) / (k + 1);
        lm = l;
        l = ln;
    }
    return l;
}

// Roots of L_n by interlacing: the roots of L_n separate those of L_{n+1}; each bracket is
// refined by bisection and polished by Newton.  Weights w_i = x_i / ((n+1) L_{n+1}(x_i))^2.
void gauss_laguerre(int n, std::vector<double>& x, std::vector<double>& w) {
    std::vector<double> prev{1.0};                        // root of L_1
    for (int deg = 2; deg <= n; ++deg) {
        std::vector<double> cur(deg);
        for (int i = 0; i < deg; ++i) {
            double lo = (i == 0) ? 0.0 : prev[i - 1];
            double hi = (i == deg - 1) ? 4.0 * deg + 3.0 : prev[i];
            double flo = laguerre(deg, lo);
            for (int it = 0; it < 200; ++it) {
                const double mid = 0.5 * (lo + hi);
                const double fm = laguerre(deg, mid);
                if ((fm < 0) == (flo < 0)) { lo = mid; flo = fm; } else { hi = mid; }
                if (hi - lo < 1e-15 * (1.0 + hi)) break;
            }
            double r = 0.5 * (lo + hi);
            for (int it = 0; it < 4; ++it) {               // Newton: L_n' = n (L_n - L_{n-1}) / x
                const double f = laguerre(deg, r), fp = deg * (f - laguerre(deg - 1, r)) / r;
                const double rn = r - f / fp;
                if (rn > lo && rn < hi) r = rn;
            }
            cur[i] = r;
        }
        prev.swap(cur);
    }
    x = prev;
    x.resize(n);
    w.resize(n);
    for (int i = 0; i < n; ++i) {
        const double l1 = laguerre(n + 1, x[i]);
        w[i] = x[i] / ((n + 1.0) * (n + 1.0) * l1 * l1);
    }
}

}  // namespace

// ================================================================================================
struct gx_grid {
    int Nx, Ny, Nz, Nl, Nm, Ns, J, nakx, naky, K, Q;
    long long nk;
    double dkx = 0, dky = 0, shat = 1;
    bool box_set = false, geo_set = false;
    bool adiabatic = false;
    bool linked = false;                        // twist-and-shift linked z operators (gx_boundary_set)
    double tau_fac = 1.0;
    double D_hyper = 0.05, f_hyp = 1.0;
    int n_hyper = 4;
    double damp_A = 0.0, damp_width = 0.125;    // end-damping layer Eq. 4.30 (off by default)
    std::vector<Species> sp;
    std::vector<double> bmag, gds2, gds21, gds22, gbdrift, gbdrift0, cvdrift, cvdrift0, bgrad, jacobian;
    bool have_lin_geo = false;
    double gradpar = 1;
    std::vector<double> xj, wj;
    std::vector<float> hT, hTinv;
    const KernelSet* ks = nullptr;
    // device
    float *dT = nullptr, *dTinv = nullptr, *dM = nullptr;
    // electromagnetic brackets (gx_nonlinear_rhs_em): (tau/Z) 2 x_j J1(alpha)/alpha table, shared plane of ones, kperp2 and
    // bmag^2 on the device, spectral chi planes, Hermite-shifted state and second result (allocated on first use)
    float *dMB = nullptr, *dones = nullptr, *dkp2 = nullptr, *dbmag2 = nullptr;
    float2 *dchis = nullptr, *dg_em = nullptr, *dout_em = nullptr;
    float2 *dtwx = nullptr, *dtwy = nullptr, *ddchi = nullptr, *dbhat = nullptr;
    unsigned* dcount = nullptr;
    int chi_buf = 0;                            // dchi buffer of the current chi planes
    unsigned* ddone = nullptr;                  // chained calls: bracket units that have finished reading dchi (all calls)
    unsigned* dchi_ready = nullptr;             // chained calls: [2][s][z][j] epoch of the call that wrote the chi plane
    bool chi_chained = false;                   // the current chi planes were written by a chained call (flags valid)
    unsigned chi_epoch = 0;                     // epoch of the chained call that wrote the current chi planes
    unsigned done_total = 0, done_at_chi = 0;   // its value once every chained call so far is done / just before the latest call with new chi planes
    unsigned* dchi_flag = nullptr;              // [s][z][j] epoch of the last call that produced the chi plane (persistent family)
    unsigned calls = 0;                         // number of gx_nonlinear_rhs calls issued (counter epoch)
    float2 *dgbuf = nullptr, *dphibuf = nullptr, *doutbuf = nullptr;   // for the *_host entry point: Hermite-block buffers each way
    unsigned* dcount_blk = nullptr;             // arrival counters of the block-wise evaluations of the *_host entry point
    cudaStream_t st_in = nullptr, st_out = nullptr, st_cmp = nullptr, st_lin = nullptr;
    cudaEvent_t ev_phi = nullptr, ev_lin = nullptr;    // gx_rhs: linear terms on st_lin under the nonlinear kernels
    cudaEvent_t ev_user = nullptr;
    cudaGraphExec_t host_graph = nullptr;       // captured pipeline of the *_host entry point for the pointers below
    const void *hg_g = nullptr, *hg_phi = nullptr, *hg_out = nullptr;
    std::vector<cudaEvent_t> ev_host;
    gx::LinTables lin;                                                  // linear-term tables
    float2* dphi_rhs = nullptr;                                         // phi of gx_rhs
    float2* static_mom = nullptr;                                       // device address of gx_static_mom on this handle's device (gx_linear_rhs_static)
    float2 *drk_y = nullptr, *drk_k = nullptr;                          // SSP-RK3 stage and slope buffers
    size_t bytes = 0, lin_bytes = 0;
    bool profile = false;
    std::vector<cudaEvent_t> ev_pool;          // 4 events per profiled call
    size_t ev_used = 0;
    std::string err;
};

// Scratch of the allocation-free entry point gx_linear_rhs_static: the Dougherty field-particle moments
// mom[s][3][z][k] (Eq. 4.14-4.18) of ONE call.  4 MiB per GPU that loads the library, held until the process exits.
// In host code `gx_static_mom` is only the host-side stand-in of the symbol, never a device address: the address is
// resolved once per device by static_mom_address() below and handed to the kernels through LinTables::mom.
constexpr size_t kStaticMomElems = GX_STATIC_SCRATCH_ELEMS;
static __device__ __align__(256) float2 gx_static_mom[kStaticMomElems];

namespace {

constexpr int kMaxDevices = 64;
std::mutex static_mom_mutex;
float2* static_mom_of_device[kMaxDevices] = {};

// Set-up time, with the handle's device current: device address of gx_static_mom on that device (cached per device).
cudaError_t static_mom_address(float2** out) {
    *out = nullptr;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(static_mom_mutex);
    if (!static_mom_of_device[dev]) {
        void* ptr = nullptr;
        e = cudaGetSymbolAddress(&ptr, gx_static_mom);
        if (e != cudaSuccess) return e;
        static_mom_of_device[dev] = (float2*)ptr;
    }
    *out = static_mom_of_device[dev];
    return cudaSuccess;
}

constexpr int kHostBufs = 3;       // Hermite-block buffers each way of gx_nonlinear_rhs_host
bool misaligned(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) != 0; }
bool overlap(const void* a, const void* b, size_t bytes) {
    const uintptr_t x = reinterpret_cast<uintptr_t>(a), y = reinterpret_cast<uintptr_t>(b);
    return x < y + bytes && y < x + bytes;
}

int fail(gx_grid* g, int code, const std::string& msg) {
    if (g) g->err = msg;
    return code;
}
int cuda_fail(gx_grid* g, cudaError_t e, const char* where) {
    return fail(g, GX_ERR_CUDA, std::string(where) + ": " + cudaGetErrorString(e));
}
#define GX_CUDA(g, call)                                            \
    do {                                                            \
        cudaError_t e_ = (call);                                    \
        if (e_ != cudaSuccess) return cuda_fail(g, e_, #call);      \
    } while (0)

template <class T> int dev_alloc(gx_grid* g, T** p, size_t n) {
    cudaError_t e = cudaMalloc((void**)p, n * sizeof(T));
    if (e != cudaSuccess) return fail(g, GX_ERR_ALLOC, std::string("cudaMalloc: ") + cudaGetErrorString(e));
    g->bytes += n * sizeof(T);
    return GX_OK;
}

bool splits(int N) {   // N = R1*R2 with R in {2,3,4,6,8,12,16}
    const int R[] = {2, 3, 4, 6, 8, 12, 16};
    for (int a : R)
        for (int b : R)
            if (a * b == N) return true;
    return false;
}

NlParams make_params(gx_grid* g, const void* gd, const void* phid, void* outd) {
    NlParams p{};
    p.g = (const float2*)gd;
    p.phi = (const float2*)phid;
    p.dchi = g->ddchi;
    p.bhat = g->dbhat;
    p.out = (float2*)outd;
    p.M = g->dM;
    p.T = g->dT;
    p.Tinv = g->dTinv;
    p.count = g->dcount;
    p.twx = g->dtwx;
    p.twy = g->dtwy;
    p.dkx = (float)g->dkx;
    p.dky = (float)g->dky;
    p.scale = (float)(1.0 / ((double)g->Nx * (double)g->Ny));
    p.Nz = g->Nz; p.Nl = g->Nl; p.Nm = g->Nm; p.Ns = g->Ns; p.J = g->J;
    if (g->ks && g->ks->family == GX_FAMILY_ROW) p.scale *= 0.5f;      // row_forward_real leaves twice the coefficients
    if (g->ks && g->ks->transposed) {
        // the kernels see x' = y, y' = x: {chi, g}' = -{chi, g}
        std::swap(p.dkx, p.dky);
        std::swap(p.twx, p.twy);
        p.scale = -p.scale;
    }
    return p;
}

long long nl_flops(const gx_grid* g) {
    // nominal FFT convention, zero columns not transformed.
    const double Nx = g->Nx, Ny = g->Ny, naky = g->naky, nk = (double)g->nk, J = g->J, Nl = g->Nl;
    const double P = (double)g->Ns * g->Nm * g->Nz * J, SZJ = (double)g->Ns * g->Nz * J;
    const double nT = 3 * P + 2 * SZJ;
    const double fft = 5 * Nx * std::log2(Nx) * naky + 2.5 * Ny * std::log2(Ny) * Nx;
    const double F = nT * fft + 3 * Nx * Ny * P + 2 * (4 * J * Nl) * nk * g->Ns * g->Nm * g->Nz +
                     (4 * nk * P + 6 * nk * SZJ);
    return (long long)F;
}

}  // namespace

// ================================================================================================
extern "C" {

int gx_grid_create(int Nx, int Ny, int Nz, int Nl, int Nm, int Ns, gx_grid** out) {
    if (!out) return GX_ERR_ARG;
    *out = nullptr;
    if (Nx < 4 || Ny < 4 || (Nx & 1) || (Ny & 1) || Nz < 1 || Nl < 1 || Nl > 16 || Nm < 1 || Ns < 1)
        return GX_ERR_ARG;
    if (!splits(Nx) || !splits(Ny)) return GX_ERR_ARG;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return GX_ERR_CUDA;
    gx_grid* g = new (std::nothrow) gx_grid();
    if (!g) return GX_ERR_ALLOC;
    g->Nx = Nx; g->Ny = Ny; g->Nz = Nz; g->Nl = Nl; g->Nm = Nm; g->Ns = Ns;
    g->K = (Nx - 1) / 3; g->Q = (Ny - 1) / 3;
    g->nakx = 2 * g->K + 1; g->naky = g->Q + 1;
    g->nk = (long long)g->nakx * g->naky;
    g->J = (3 * Nl - 1) / 2;
    g->sp.resize(Ns);
    g->adiabatic = (Ns == 1);
    g->ks = find_set(Nx, Ny);
    *out = g;                       // returned even on failure below so that gx_last_error works
    if (!g->ks) return fail(g, GX_ERR_UNSUPPORTED, "no kernel instantiation for this (Nx,Ny)");
    GX_CUDA(g, g->ks->prepare());      // per device and per handle: no process-wide cache of function attributes
    GX_CUDA(g, gx::lin_prepare());
    GX_CUDA(g, static_mom_address(&g->static_mom));      // set-up for gx_linear_rhs_static (nothing allocated)

    gauss_laguerre(g->J, g->xj, g->wj);
    g->hT.resize((size_t)g->J * Nl);
    g->hTinv.resize((size_t)Nl * g->J);
    for (int j = 0; j < g->J; ++j)
        for (int l = 0; l < Nl; ++l) {
            const double psi = ((l & 1) ? -1.0 : 1.0) * laguerre(l, g->xj[j]);   // psi_l = (-1)^l L_l
            g->hT[(size_t)j * Nl + l] = (float)psi;
            g->hTinv[(size_t)l * g->J + j] = (float)(g->wj[j] * psi);
        }
    int rc;
    if ((rc = dev_alloc(g, &g->dT, g->hT.size()))) return rc;
    if ((rc = dev_alloc(g, &g->dTinv, g->hTinv.size()))) return rc;
    GX_CUDA(g, cudaMemcpy(g->dT, g->hT.data(), g->hT.size() * sizeof(float), cudaMemcpyHostToDevice));
    GX_CUDA(g, cudaMemcpy(g->dTinv, g->hTinv.data(), g->hTinv.size() * sizeof(float), cudaMemcpyHostToDevice));

    std::vector<float2> tw(Nx);
    for (int t = 0; t < Nx; ++t) {
        const double a = 2.0 * M_PI * t / Nx;
        tw[t] = make_float2((float)std::cos(a), (float)std::sin(a));
    }
    if ((rc = dev_alloc(g, &g->dtwx, (size_t)Nx))) return rc;
    GX_CUDA(g, cudaMemcpy(g->dtwx, tw.data(), Nx * sizeof(float2), cudaMemcpyHostToDevice));
    tw.resize(Ny);
    for (int t = 0; t < Ny; ++t) {
        const double a = 2.0 * M_PI * t / Ny;
        tw[t] = make_float2((float)std::cos(a), (float)std::sin(a));
    }
    if ((rc = dev_alloc(g, &g->dtwy, (size_t)Ny))) return rc;
    GX_CUDA(g, cudaMemcpy(g->dtwy, tw.data(), Ny * sizeof(float2), cudaMemcpyHostToDevice));

    const size_t szj = (size_t)Ns * Nz * g->J;
    if ((rc = dev_alloc(g, &g->dM, szj * g->nk))) return rc;
    if ((rc = dev_alloc(g, &g->ddchi, 2 * szj * Nx * Ny))) return rc;     // two buffers: chi of call N+1 under the tail of call N
    if ((rc = dev_alloc(g, &g->dbhat, szj * Nm * g->nk))) return rc;
    if ((rc = dev_alloc(g, &g->dcount, (size_t)Ns * Nm * Nz))) return rc;
    GX_CUDA(g, cudaMemset(g->dcount, 0, (size_t)Ns * Nm * Nz * sizeof(unsigned)));
    if ((rc = dev_alloc(g, &g->dchi_ready, 2 * szj))) return rc;
    GX_CUDA(g, cudaMemset(g->dchi_ready, 0, 2 * szj * sizeof(unsigned)));
    if ((rc = dev_alloc(g, &g->ddone, 4))) return rc;
    GX_CUDA(g, cudaMemset(g->ddone, 0, 4 * sizeof(unsigned)));
    if ((rc = dev_alloc(g, &g->dchi_flag, szj))) return rc;
    GX_CUDA(g, cudaMemset(g->dchi_flag, 0, szj * sizeof(unsigned)));
    return GX_OK;
}

int gx_grid_destroy(gx_grid* g) {
    if (!g) return GX_ERR_ARG;
    cudaFree(g->dT); cudaFree(g->dTinv); cudaFree(g->dM); cudaFree(g->dMB); cudaFree(g->dones); cudaFree(g->dkp2);
    cudaFree(g->dbmag2); cudaFree(g->dchis); cudaFree(g->dg_em); cudaFree(g->dout_em); cudaFree(g->dtwx); cudaFree(g->dtwy);
    cudaFree(g->ddchi); cudaFree(g->dbhat); cudaFree(g->dcount); cudaFree(g->ddone); cudaFree(g->dchi_ready); cudaFree(g->dchi_flag); cudaFree(g->dgbuf); cudaFree(g->dphibuf); cudaFree(g->doutbuf);
    cudaFree(g->dphi_rhs); cudaFree(g->drk_y); cudaFree(g->drk_k);
    for (auto e : g->ev_pool) cudaEventDestroy(e);
    for (auto e : g->ev_host) cudaEventDestroy(e);
    if (g->host_graph) cudaGraphExecDestroy(g->host_graph);
    if (g->st_in) cudaStreamDestroy(g->st_in);
    if (g->st_cmp) cudaStreamDestroy(g->st_cmp);
    if (g->st_lin) cudaStreamDestroy(g->st_lin);
    if (g->ev_phi) cudaEventDestroy(g->ev_phi);
    if (g->ev_lin) cudaEventDestroy(g->ev_lin);
    if (g->ev_user) cudaEventDestroy(g->ev_user);
    if (g->st_out) cudaStreamDestroy(g->st_out);
    cudaFree(g->dcount_blk);
    gx::lin_tables_free(g->lin);
    delete g;
    return GX_OK;
}

int gx_box_set(gx_grid* g, double dky, double dkx, double shat) {
    if (!g) return GX_ERR_ARG;
    if (!(dky > 0) || !(dkx > 0) || shat == 0.0) return fail(g, GX_ERR_ARG, "gx_box_set: dky, dkx > 0, shat != 0");
    g->dky = dky; g->dkx = dkx; g->shat = shat;
    g->box_set = true;
    g->geo_set = false;
    return GX_OK;
}

int gx_species_set(gx_grid* g, int s, double Z, double mass, double temp, double dens, double tprim,
                   double fprim, double nu_ss) {
    if (!g) return GX_ERR_ARG;
    if (s < 0 || s >= g->Ns || Z == 0.0 || mass < 0 || !(temp > 0) || !(dens > 0))
        return fail(g, GX_ERR_ARG, "gx_species_set: bad argument");
    Species& sp = g->sp[s];
    sp.Z = Z; sp.mass = mass; sp.temp = temp; sp.dens = dens; sp.tprim = tprim; sp.fprim = fprim; sp.nu = nu_ss;
    sp.set = true;
    g->geo_set = false;
    return GX_OK;
}

int gx_adiabatic_set(gx_grid* g, int enabled, double tau_fac) {
    if (!g) return GX_ERR_ARG;
    if (enabled && g->Ns != 1) return fail(g, GX_ERR_ARG, "adiabatic electrons need Ns == 1");
    g->adiabatic = enabled != 0;
    g->tau_fac = tau_fac;
    g->geo_set = false;
    return GX_OK;
}

int gx_boundary_set(gx_grid* g, int linked) {
    if (!g) return GX_ERR_ARG;
    g->linked = linked != 0;
    g->geo_set = false;
    return GX_OK;
}

int gx_dissipation_set(gx_grid* g, double D_hyper, int n_hyper, double f_hyp) {
    if (!g) return GX_ERR_ARG;
    if (D_hyper < 0 || n_hyper < 0 || f_hyp < 0) return fail(g, GX_ERR_ARG, "negative dissipation parameter");
    g->D_hyper = D_hyper; g->n_hyper = n_hyper; g->f_hyp = f_hyp;
    g->geo_set = false;
    return GX_OK;
}

int gx_damping_set(gx_grid* g, double A, double width_fraction) {
    if (!g) return GX_ERR_ARG;
    if (A < 0 || !(width_fraction > 0) || width_fraction > 0.5) return fail(g, GX_ERR_ARG, "gx_damping_set: A >= 0, 0 < width_fraction <= 1/2");
    g->damp_A = A; g->damp_width = width_fraction;
    g->geo_set = false;
    return GX_OK;
}

int gx_geometry_set(gx_grid* g, const double* bmag, const double* gds2, const double* gds21,
                    const double* gds22, const double* gbdrift, const double* gbdrift0,
                    const double* cvdrift, const double* cvdrift0, const double* bgrad,
                    const double* jacobian, double gradpar) {
    if (!g) return GX_ERR_ARG;
    if (!g->ks) return fail(g, GX_ERR_UNSUPPORTED, "no kernel instantiation for this (Nx,Ny)");
    if (!bmag || !gds2 || !gds21 || !gds22) return fail(g, GX_ERR_ARG, "gx_geometry_set: null metric array");
    if (!g->box_set) return fail(g, GX_ERR_STATE, "gx_geometry_set: call gx_box_set first");
    for (const auto& s : g->sp)
        if (!s.set) return fail(g, GX_ERR_STATE, "gx_geometry_set: call gx_species_set for every species first");
    const int Nz = g->Nz;
    g->bmag.assign(bmag, bmag + Nz); g->gds2.assign(gds2, gds2 + Nz);
    g->gds21.assign(gds21, gds21 + Nz); g->gds22.assign(gds22, gds22 + Nz);
    g->have_lin_geo = gbdrift && gbdrift0 && cvdrift && cvdrift0 && bgrad && jacobian;
    if (g->have_lin_geo) {
        g->gbdrift.assign(gbdrift, gbdrift + Nz); g->gbdrift0.assign(gbdrift0, gbdrift0 + Nz);
        g->cvdrift.assign(cvdrift, cvdrift + Nz); g->cvdrift0.assign(cvdrift0, cvdrift0 + Nz);
        g->bgrad.assign(bgrad, bgrad + Nz); g->jacobian.assign(jacobian, jacobian + Nz);
    }
    g->gradpar = gradpar;
    for (int z = 0; z < Nz; ++z)
        if (!(bmag[z] > 0)) return fail(g, GX_ERR_ARG, "gx_geometry_set: bmag must be positive");

    // gyroaverage table M[s][z][j][kx][ky] = J0( sqrt(2 x_j b_s) ), b_s = kperp2 tau m / (Z^2 bmag^2)
    // (PAPER.md line 85), kperp2 = ky^2 gds2 + 2 kx ky gds21/shat + kx^2 gds22/shat^2 (lines 681-686).
    const int nakx = g->nakx, naky = g->naky, J = g->J, K = g->K;
    std::vector<float> M((size_t)g->Ns * Nz * J * g->nk);
    std::vector<double> kp2((size_t)Nz * g->nk);
    for (int z = 0; z < Nz; ++z)
        for (int i = 0; i < nakx; ++i) {
            const double kx = g->dkx * (i <= K ? i : i - nakx);
            for (int q = 0; q < naky; ++q) {
                const double ky = g->dky * q;
                kp2[((size_t)z * nakx + i) * naky + q] = ky * ky * gds2[z] + 2.0 * kx * ky * gds21[z] / g->shat +
                                                          kx * kx * gds22[z] / (g->shat * g->shat);
            }
        }
    for (int s = 0; s < g->Ns; ++s) {
        const Species& sp = g->sp[s];
        const double rho2 = sp.temp * sp.mass / (sp.Z * sp.Z);
        for (int z = 0; z < Nz; ++z) {
            const double fac = rho2 / (bmag[z] * bmag[z]);
            for (int j = 0; j < J; ++j) {
                float* Mp = M.data() + (((size_t)s * Nz + z) * J + j) * g->nk;
                const double* kp = kp2.data() + (size_t)z * g->nk;
                for (long long k = 0; k < g->nk; ++k) {
                    const double b = kp[k] * fac;
                    Mp[k] = (float)::j0(std::sqrt(2.0 * g->xj[j] * (b > 0 ? b : 0.0)));
                }
            }
        }
    }
    GX_CUDA(g, cudaMemcpy(g->dM, M.data(), M.size() * sizeof(float), cudaMemcpyHostToDevice));
    {   // electromagnetic tables (row f4): MB[s][z][j][k] = (tau/Z) 2 x_j J1(alpha)/alpha (Eq. 4.5), kperp2, bmag^2
        std::vector<float> MB(M.size()), kf(kp2.size()), b2(Nz);
        for (int s = 0; s < g->Ns; ++s) {
            const Species& sp = g->sp[s];
            const double rho2 = sp.temp * sp.mass / (sp.Z * sp.Z), tz = sp.temp / sp.Z;
            for (int z = 0; z < Nz; ++z)
                for (int j = 0; j < J; ++j) {
                    float* Mp = MB.data() + (((size_t)s * Nz + z) * J + j) * g->nk;
                    const double* kp = kp2.data() + (size_t)z * g->nk;
                    for (long long k = 0; k < g->nk; ++k) {
                        const double b = std::max(0.0, kp[k] * rho2 / (bmag[z] * bmag[z]));
                        const double a = std::sqrt(2.0 * g->xj[j] * b);
                        const double r = a > 1e-8 ? ::j1(a) / a : 0.5 - a * a / 16.0;
                        Mp[k] = (float)(tz * 2.0 * g->xj[j] * r);
                    }
                }
        }
        for (size_t i = 0; i < kp2.size(); ++i) kf[i] = (float)kp2[i];
        for (int z = 0; z < Nz; ++z) b2[z] = (float)(bmag[z] * bmag[z]);
        int rc;
        if (!g->dMB) {
            if ((rc = dev_alloc(g, &g->dMB, MB.size()))) return rc;
            if ((rc = dev_alloc(g, &g->dkp2, kf.size()))) return rc;
            if ((rc = dev_alloc(g, &g->dbmag2, b2.size()))) return rc;
            if ((rc = dev_alloc(g, &g->dones, (size_t)g->nk))) return rc;
            std::vector<float> ones((size_t)g->nk, 1.f);
            GX_CUDA(g, cudaMemcpy(g->dones, ones.data(), ones.size() * sizeof(float), cudaMemcpyHostToDevice));
        }
        GX_CUDA(g, cudaMemcpy(g->dMB, MB.data(), MB.size() * sizeof(float), cudaMemcpyHostToDevice));
        GX_CUDA(g, cudaMemcpy(g->dkp2, kf.data(), kf.size() * sizeof(float), cudaMemcpyHostToDevice));
        GX_CUDA(g, cudaMemcpy(g->dbmag2, b2.data(), b2.size() * sizeof(float), cudaMemcpyHostToDevice));
    }

    if (g->have_lin_geo) {
        gx::LinHostInput in;
        in.Nz = Nz; in.Nl = g->Nl; in.Nm = g->Nm; in.Ns = g->Ns; in.nakx = nakx; in.naky = naky;
        in.dkx = g->dkx; in.dky = g->dky; in.shat = g->shat; in.gradpar = gradpar;
        in.kp2 = kp2.data(); in.bmag = g->bmag.data(); in.gbdrift = g->gbdrift.data();
        in.gbdrift0 = g->gbdrift0.data(); in.cvdrift = g->cvdrift.data(); in.cvdrift0 = g->cvdrift0.data();
        in.bgrad = g->bgrad.data(); in.jacobian = g->jacobian.data();
        in.adiabatic = g->adiabatic; in.tau_fac = g->tau_fac;
        in.D_hyper = g->D_hyper; in.n_hyper = g->n_hyper; in.f_hyp = g->f_hyp;
        in.linked = g->linked;
        in.damp_A = g->damp_A; in.damp_width = g->damp_width;
        for (const auto& sp : g->sp)
            in.species.push_back({sp.Z, sp.mass, sp.temp, sp.dens, sp.tprim, sp.fprim, sp.nu});
        std::string msg;
        size_t bytes = 0;
        if (!gx::lin_tables_build(in, g->lin, bytes, msg))
            return fail(g, msg.find("quantised") != std::string::npos ? GX_ERR_ARG : GX_ERR_CUDA, msg);
        g->bytes += bytes - g->lin_bytes;          // a rebuilt table replaces the old one
        g->lin_bytes = bytes;
        if (!g->dphi_rhs) {
            int rc = dev_alloc(g, &g->dphi_rhs, (size_t)Nz * g->nk);
            if (rc) return rc;
        }
    }
    if (g->host_graph) { cudaGraphExecDestroy(g->host_graph); g->host_graph = nullptr; }   // table pointers may have changed
    g->geo_set = true;
    return GX_OK;
}

}  // extern "C"

namespace {
// Enqueues the kernels of one evaluation for Nm_eff Hermite moments (p.Nm = Nm_eff; the arrays behind p.g / p.out
// hold exactly those moments).  do_chi = false reuses the chi planes already in the workspace (same phi).
// count / calls: arrival counters of the separate inverse-Laguerre kernel and their epoch.
int nl_enqueue(gx_grid* g, NlParams p, int Nm_eff, bool do_chi, unsigned* count, unsigned* calls, cudaStream_t st,
               cudaEvent_t* ev, cudaEvent_t before_out = nullptr) {
    // before_out: event the stream waits for before the kernel that writes `out` (separate inverse-Laguerre kernel only)
    // calls == nullptr: the counters are zeroed by a memset node before the kernels and the target is J itself
    // (no epoch in the kernel arguments: the sequence can be captured in a CUDA graph and replayed)
    p.Nm = Nm_eff;
    p.count = count;
    const int szj = g->Ns * g->Nz * g->J;
    if (calls) {
        // the kernels take the call's epoch as an argument: a caller's CUDA graph would replay stale epochs
        cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
        if (cudaStreamIsCapturing(st, &cs) == cudaSuccess && cs != cudaStreamCaptureStatusNone)
            return fail(g, GX_ERR_STATE, "the compute calls cannot be recorded into a CUDA graph (gx_nonlinear_rhs_host replays its own)");
    }
    if (do_chi) g->chi_buf ^= 1;
    p.dchi = g->ddchi + (size_t)g->chi_buf * szj * g->Nx * g->Ny;
    // a8 inside the bracket kernel (last node unit of an (s,m,z) to arrive) unless out already holds the linear terms
    const bool fuse_a8 = g->ks->closer && g->J <= 5 && g->Nl <= 4 && !before_out && !p.accumulate && std::getenv("GX_A8_KERNEL") == nullptr;
    p.ZG = 1;
    if (fuse_a8)                               // spacing between the J node units of an (s,m,z): only the closer needs it
        for (int c = 2; c <= 4; ++c)
            if (g->Nz % c == 0) p.ZG = c;
    if (const char* e = std::getenv("GX_ZG")) { const int c = std::atoi(e); if (c >= 1 && g->Nz % c == 0) p.ZG = c; }
    if (!calls && !g->ks->fused_laguerre)
        GX_CUDA(g, cudaMemsetAsync(count, 0, (size_t)g->Ns * Nm_eff * g->Nz * sizeof(unsigned), st));
    if (g->ks->launch_call) {
        g->calls += 1;
        if (ev) GX_CUDA(g, cudaEventRecord(ev[1], st));
        GX_CUDA(g, g->ks->launch_call(p, g->dchi_flag, g->calls, szj + szj * Nm_eff, st));
        if (ev) { GX_CUDA(g, cudaEventRecord(ev[2], st)); GX_CUDA(g, cudaEventRecord(ev[3], st)); }
        return GX_OK;
    }
    // Outside graph capture (calls != nullptr) the chi grid carries the PDL attribute: after a call whose last kernel
    // is the bracket grid it starts while that grid's last wave still runs.  A foreign kernel in front of it never
    // triggers early, so phi / g written by the caller's own kernels are complete before the chi grid starts.
    unsigned target = (unsigned)g->J;
    if (!g->ks->fused_laguerre && calls) { *calls += 1; target = *calls * (unsigned)g->J; }
    p.a8_target = fuse_a8 ? target : 0u;
    // GX_CLUSTER=1: a8 over the distributed shared memory of a J-CTA cluster instead of the closer.  Measured slower
    // (Cyclone 64.4 against 56.7 us per call: co-scheduling of 5 CTAs and two cluster barriers per unit), kept as an option.
    p.cluster = (fuse_a8 && g->J <= 8 && std::getenv("GX_CLUSTER") != nullptr) ? 1 : 0;
    // (a call that reuses chi planes is chained only if the chained flags describe those planes)
    // Calls with the separate inverse-Laguerre kernel (gx_rhs) are not chained: that kernel never triggers early.
    const bool chained = calls && fuse_a8 && g->ks->launch_chi_pdl && std::getenv("GX_CHI_SERIAL") == nullptr && (do_chi || g->chi_chained);
    if (do_chi) g->chi_chained = chained;
    if (chained) {
        // Counters instead of grid-completion order (nl_row_kernels.cuh): the chi grid of this call writes the dchi
        // buffer that was read by the calls before the latest one with new chi planes; all their units have left the
        // row phase once done reaches the total recorded just before that call (wrap-safe sequence arithmetic).
        p.done = g->ddone;
        if (do_chi) { p.chi_need = g->done_at_chi; g->done_at_chi = g->done_total; g->chi_epoch = *calls; }
        g->done_total += (unsigned)(szj * Nm_eff);
        p.chi_ready = g->dchi_ready + (size_t)g->chi_buf * szj;
        p.chi_epoch = g->chi_epoch;
    }
    if (do_chi) {
        auto chi = !chained ? g->ks->launch_chi
                            : (std::getenv("GX_CHI_WIDE") && g->ks->launch_chi_pdl_wide ? g->ks->launch_chi_pdl_wide : g->ks->launch_chi_pdl);
        GX_CUDA(g, chi(p, szj, st));
    }
    if (ev) GX_CUDA(g, cudaEventRecord(ev[1], st));
    GX_CUDA(g, g->ks->launch_bracket(p, szj * Nm_eff, st));
    if (ev) GX_CUDA(g, cudaEventRecord(ev[2], st));
    if (!g->ks->fused_laguerre && !fuse_a8) {
        const int vec = (g->nk % 2 == 0) ? 2 : 1;
        const int nkv = (int)(g->nk / vec);
        dim3 grid((unsigned)((nkv + 255) / 256), (unsigned)(g->Ns * Nm_eff * g->Nz));
        const int nk = (int)g->nk;
        if (before_out) GX_CUDA(g, cudaStreamWaitEvent(st, before_out, 0));
        cudaError_t e;
        const int mode = p.st_out ? 2 : (p.accumulate ? 1 : 0);
#define GX_LAGINV_M(L, J, M)                                                                                      \
    e = (vec == 2) ? launch_pdl(gx::laguerre_inverse_kernel<L, J, 2, M>, grid, dim3(256), 0, st, p, nk, target)  \
                   : launch_pdl(gx::laguerre_inverse_kernel<L, J, 1, M>, grid, dim3(256), 0, st, p, nk, target)
#define GX_LAGINV(L, J)                                                                  \
    do {                                                                                 \
        if (mode == 2) GX_LAGINV_M(L, J, 2);                                            \
        else if (mode == 1) GX_LAGINV_M(L, J, 1);                                       \
        else GX_LAGINV_M(L, J, 0);                                                      \
    } while (0)
        if (g->Nl <= 4) GX_LAGINV(4, 5);
        else if (g->Nl <= 8) GX_LAGINV(8, 11);
        else GX_LAGINV(16, 23);
#undef GX_LAGINV
#undef GX_LAGINV_M
        GX_CUDA(g, e);
    }
    if (ev) GX_CUDA(g, cudaEventRecord(ev[3], st));
    return GX_OK;
}
}  // namespace

extern "C" {

int gx_nonlinear_rhs(gx_grid* g, const void* g_dev, const void* phi_dev, void* out_dev, void* cuda_stream) {
    if (!g) return GX_ERR_ARG;
    if (!g_dev || !phi_dev || !out_dev) return fail(g, GX_ERR_ARG, "gx_nonlinear_rhs: null pointer");
    const size_t gbytes = (size_t)g->Ns * g->Nm * g->Nl * g->Nz * g->nk * sizeof(float2);
    if (overlap(g_dev, out_dev, gbytes)) return fail(g, GX_ERR_ARG, "gx_nonlinear_rhs: out must not alias g");
    if (misaligned(g_dev) || misaligned(phi_dev) || misaligned(out_dev))
        return fail(g, GX_ERR_ARG, "gx_nonlinear_rhs: device pointers must be 16-byte aligned");
    if (!g->ks) return fail(g, GX_ERR_UNSUPPORTED, "no kernel instantiation for this (Nx,Ny)");
    if (!g->geo_set) return fail(g, GX_ERR_STATE, "gx_nonlinear_rhs: geometry not set");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const NlParams p = make_params(g, g_dev, phi_dev, out_dev);
    cudaEvent_t* ev = nullptr;
    if (g->profile) {
        if (g->ev_used + 4 > g->ev_pool.size()) {
            const size_t old = g->ev_pool.size();
            g->ev_pool.resize(old + 4 * 256);
            for (size_t i = old; i < g->ev_pool.size(); ++i) GX_CUDA(g, cudaEventCreate(&g->ev_pool[i]));
        }
        ev = &g->ev_pool[g->ev_used];
        g->ev_used += 4;
        GX_CUDA(g, cudaEventRecord(ev[0], st));
    }
    return nl_enqueue(g, p, g->Nm, true, g->dcount, &g->calls, st, ev);
}

int gx_nonlinear_rhs_em(gx_grid* g, const void* g_dev, const void* phi_dev, const void* apar_dev, const void* bpar_dev,
                        void* out_dev, void* cuda_stream) {
    if (!g) return GX_ERR_ARG;
    if (!g_dev || !phi_dev || !apar_dev || !bpar_dev || !out_dev) return fail(g, GX_ERR_ARG, "gx_nonlinear_rhs_em: null pointer");
    const size_t ng = (size_t)g->Ns * g->Nm * g->Nl * g->Nz * g->nk;
    if (overlap(g_dev, out_dev, ng * sizeof(float2))) return fail(g, GX_ERR_ARG, "gx_nonlinear_rhs_em: out must not alias g");
    if (misaligned(g_dev) || misaligned(phi_dev) || misaligned(apar_dev) || misaligned(bpar_dev) || misaligned(out_dev))
        return fail(g, GX_ERR_ARG, "gx_nonlinear_rhs_em: device pointers must be 16-byte aligned");
    if (!g->ks) return fail(g, GX_ERR_UNSUPPORTED, "no kernel instantiation for this (Nx,Ny)");
    if (!g->geo_set || !g->have_lin_geo) return fail(g, GX_ERR_STATE, "gx_nonlinear_rhs_em: full geometry not set");
    if (ng % 2) return fail(g, GX_ERR_UNSUPPORTED, "gx_nonlinear_rhs_em: odd number of coefficients");
    const size_t szj = (size_t)g->Ns * g->Nz * g->J;
    int rc;
    if (!g->dchis) {
        if ((rc = dev_alloc(g, &g->dchis, szj * g->nk))) return rc;
        if ((rc = dev_alloc(g, &g->dg_em, ng))) return rc;
        if ((rc = dev_alloc(g, &g->dout_em, ng))) return rc;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const dim3 cgrid((unsigned)((g->nk + 255) / 256), (unsigned)szj);
    // out = -L F{ J0 Phi + (tau/Z) 2 muB (J1/alpha) dB_par/B , gt_m }            (D1 lines 1 and 4)
    gx::em_chi_spectral_kernel<<<cgrid, 256, 0, st>>>(g->dM, g->dMB, (const float2*)phi_dev, (const float2*)bpar_dev, g->dchis,
                                                      (int)g->nk, g->Nz, g->J);
    NlParams p = make_params(g, g_dev, g->dchis, out_dev);
    p.M = g->dones; p.phi_by_unit = 1; p.M_shared = 1;
    if ((rc = nl_enqueue(g, p, g->Nm, true, g->dcount, &g->calls, st, nullptr))) return rc;
    // out += -L F{ J0 A_par , gt2_m },  G2_{l,m} = -v_ts ( sqrt(m+1) G_{l,m+1} + sqrt(m) G_{l,m-1} )   (D1 lines 2-3)
    gx::em_chi_spectral_kernel<<<cgrid, 256, 0, st>>>(g->dM, nullptr, (const float2*)apar_dev, nullptr, g->dchis, (int)g->nk, g->Nz, g->J);
    {
        const unsigned pl = (unsigned)((size_t)g->Nl * g->Nz * g->nk);
        gx::em_hermite_shift_kernel<<<dim3((pl + 255) / 256, (unsigned)(g->Ns * g->Nm)), 256, 0, st>>>(g->lin, (const float2*)g_dev, g->dg_em);
    }
    p = make_params(g, g->dg_em, g->dchis, g->dout_em);
    p.M = g->dones; p.phi_by_unit = 1; p.M_shared = 1;
    if ((rc = nl_enqueue(g, p, g->Nm, true, g->dcount, &g->calls, st, nullptr))) return rc;
    gx::em_add_kernel<<<(unsigned)((ng / 2 + 255) / 256), 256, 0, st>>>((float4*)out_dev, (const float4*)g->dout_em, ng / 2);
    GX_CUDA(g, cudaGetLastError());
    return GX_OK;
}

int gx_field_solve_em(gx_grid* g, const void* g_dev, double beta, void* phi_dev, void* apar_dev, void* bpar_dev, void* cuda_stream) {
    if (!g) return GX_ERR_ARG;
    if (!g_dev || !phi_dev || !apar_dev || !bpar_dev || beta < 0) return fail(g, GX_ERR_ARG, "gx_field_solve_em: null pointer or beta < 0");
    if (!g->geo_set || !g->have_lin_geo) return fail(g, GX_ERR_STATE, "gx_field_solve_em: full geometry not set");
    gx::EmSpecies e{};
    for (int s = 0; s < g->Ns; ++s) {
        const Species& sp = g->sp[s];
        e.qn[s] = (float)(sp.Z * sp.dens);
        e.z2nt[s] = (float)(sp.Z * sp.Z * sp.dens / sp.temp);
        e.nt[s] = (float)(sp.dens * sp.temp);
        e.z2nm[s] = (float)(sp.Z * sp.Z * sp.dens / sp.mass);
        e.qnv[s] = (float)(sp.Z * sp.dens * std::sqrt(sp.temp / sp.mass));
    }
    dim3 grid((unsigned)((g->nk + 255) / 256), (unsigned)g->Nz);
    gx::field_solve_em_kernel<<<grid, 256, 0, (cudaStream_t)cuda_stream>>>(g->lin, e, g->dkp2, g->dbmag2, (float)beta, (const float2*)g_dev,
                                                                           (float2*)phi_dev, (float2*)apar_dev, (float2*)bpar_dev);
    GX_CUDA(g, cudaGetLastError());
    return GX_OK;
}

int gx_profile_set(gx_grid* g, int enabled) {
    if (!g) return GX_ERR_ARG;
    g->profile = enabled != 0;
    return GX_OK;
}

int gx_profile_get(gx_grid* g, double* ms, long long* calls) {
    if (!g || !ms || !calls) return GX_ERR_ARG;
    *calls = (long long)(g->ev_used / 4);
    for (size_t c = 0; c < g->ev_used; c += 4) {
        GX_CUDA(g, cudaEventSynchronize(g->ev_pool[c + 3]));
        for (int k = 0; k < 3; ++k) {
            float t = 0.f;
            GX_CUDA(g, cudaEventElapsedTime(&t, g->ev_pool[c + k], g->ev_pool[c + k + 1]));
            ms[k] += t;
        }
    }
    g->ev_used = 0;
    return GX_OK;
}

int gx_nonlinear_rhs_host(gx_grid* g, const void* g_host, const void* phi_host, void* out_host, void* cuda_stream) {
    if (!g) return GX_ERR_ARG;
    if (!g_host || !phi_host || !out_host) return fail(g, GX_ERR_ARG, "gx_nonlinear_rhs_host: null pointer");
    if (!g->ks) return fail(g, GX_ERR_UNSUPPORTED, "no kernel instantiation for this (Nx,Ny)");
    if (!g->geo_set) return fail(g, GX_ERR_STATE, "gx_nonlinear_rhs_host: geometry not set");
    const size_t per_m = (size_t)g->Nl * g->Nz * g->nk, np = (size_t)g->Nz * g->nk;
    // Hermite blocks: the term is diagonal in m, so block b of every species is an independent sub-problem that
    // shares the chi planes.  Three streams: H2D of block b+1 and D2H of block b-1 overlap the kernels of block b
    // (the PCIe link is full duplex); three block buffers each way.
    const bool pipelined = g->ks->launch_call == nullptr && g->Nm > 1;
    int want = 4;       // about four blocks: each is one launch-latency-bound wave of kernels (GX_HOST_BLOCKS overrides)
    if (const char* e = std::getenv("GX_HOST_BLOCKS")) want = std::max(1, std::atoi(e));
    const int mb = pipelined ? std::max(1, (g->Nm + want - 1) / want) : g->Nm;      // moments per block
    const int nb = (g->Nm + mb - 1) / mb;
    const size_t blk = (size_t)g->Ns * mb * per_m;
    int rc;
    if (!g->dgbuf) {
        if ((rc = dev_alloc(g, &g->dgbuf, kHostBufs * blk))) return rc;
        if ((rc = dev_alloc(g, &g->doutbuf, kHostBufs * blk))) return rc;
        if ((rc = dev_alloc(g, &g->dphibuf, np))) return rc;
        if ((rc = dev_alloc(g, &g->dcount_blk, (size_t)g->Ns * mb * g->Nz))) return rc;
        GX_CUDA(g, cudaMemset(g->dcount_blk, 0, (size_t)g->Ns * mb * g->Nz * sizeof(unsigned)));
        GX_CUDA(g, cudaStreamCreateWithFlags(&g->st_cmp, cudaStreamNonBlocking));
        GX_CUDA(g, cudaEventCreateWithFlags(&g->ev_user, cudaEventDisableTiming));
        GX_CUDA(g, cudaStreamCreateWithFlags(&g->st_in, cudaStreamNonBlocking));
        GX_CUDA(g, cudaStreamCreateWithFlags(&g->st_out, cudaStreamNonBlocking));
        g->ev_host.resize(3 * 64 + 2);
        for (auto& e : g->ev_host) GX_CUDA(g, cudaEventCreateWithFlags(&e, std::getenv("GX_HOST_TRACE") ? cudaEventDefault : cudaEventDisableTiming));
    }
    if (nb > 64) return fail(g, GX_ERR_UNSUPPORTED, "gx_nonlinear_rhs_host: more than 64 Hermite blocks");
    // all work runs on three internal streams (the caller's stream may be the legacy default stream, which cannot
    // be captured); it is ordered after the work already queued on the caller's stream, and the call synchronises
    cudaStream_t ust = (cudaStream_t)cuda_stream, st = g->st_cmp, sin = g->st_in, sout = g->st_out;
    GX_CUDA(g, cudaEventRecord(g->ev_user, ust));
    GX_CUDA(g, cudaStreamWaitEvent(st, g->ev_user, 0));
    // The whole pipeline (about a hundred copies, launches and event edges) is captured once per set of host
    // pointers into a CUDA graph and replayed: one launch per call instead of a hundred driver calls.
    const bool use_graph = pipelined && std::getenv("GX_HOST_NO_GRAPH") == nullptr;
    if (use_graph && g->host_graph && g->hg_g == g_host && g->hg_phi == phi_host && g->hg_out == out_host) {
        GX_CUDA(g, cudaGraphLaunch(g->host_graph, st));
        GX_CUDA(g, cudaStreamSynchronize(st));
        return GX_OK;
    }
    if (use_graph) {
        if (g->host_graph) { cudaGraphExecDestroy(g->host_graph); g->host_graph = nullptr; }
        GX_CUDA(g, cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal));
    }
    const float2* gh = (const float2*)g_host;
    float2* oh = (float2*)out_host;
    cudaEvent_t* e_in = g->ev_host.data();          // block copied in
    cudaEvent_t* e_cmp = e_in + 64;                 // block computed
    cudaEvent_t* e_out = e_cmp + 64;                // block copied out
    cudaEvent_t e_start = g->ev_host[3 * 64], e_phi = g->ev_host[3 * 64 + 1];
    GX_CUDA(g, cudaEventRecord(e_start, st));       // work already queued on the caller's stream comes first
    GX_CUDA(g, cudaStreamWaitEvent(sin, e_start, 0));
    GX_CUDA(g, cudaStreamWaitEvent(sout, e_start, 0));
    GX_CUDA(g, cudaMemcpyAsync(g->dphibuf, phi_host, np * sizeof(float2), cudaMemcpyHostToDevice, sin));
    GX_CUDA(g, cudaEventRecord(e_phi, sin));
    GX_CUDA(g, cudaStreamWaitEvent(st, e_phi, 0));
    for (int b = 0; b < nb; ++b) {
        const int m0 = b * mb, nm = std::min(mb, g->Nm - m0);
        float2* dg = g->dgbuf + (size_t)(b % kHostBufs) * blk;
        float2* dout = g->doutbuf + (size_t)(b % kHostBufs) * blk;
        if (b >= kHostBufs) GX_CUDA(g, cudaStreamWaitEvent(sin, e_cmp[b - kHostBufs], 0));       // block buffer free again
        for (int s = 0; s < g->Ns; ++s)
            GX_CUDA(g, cudaMemcpyAsync(dg + (size_t)s * nm * per_m, gh + ((size_t)s * g->Nm + m0) * per_m,
                                       (size_t)nm * per_m * sizeof(float2), cudaMemcpyHostToDevice, sin));
        GX_CUDA(g, cudaEventRecord(e_in[b], sin));
        GX_CUDA(g, cudaStreamWaitEvent(st, e_in[b], 0));
        if (b >= kHostBufs) GX_CUDA(g, cudaStreamWaitEvent(st, e_out[b - kHostBufs], 0));        // its result has left the device
        const NlParams p = make_params(g, dg, g->dphibuf, dout);
        if (pipelined) rc = nl_enqueue(g, p, nm, b == 0, g->dcount_blk, nullptr, st, nullptr);
        else rc = nl_enqueue(g, p, nm, true, g->dcount, &g->calls, st, nullptr);
        if (rc) {
            if (use_graph) { cudaGraph_t dead = nullptr; cudaStreamEndCapture(st, &dead); if (dead) cudaGraphDestroy(dead); }
            return rc;
        }
        GX_CUDA(g, cudaEventRecord(e_cmp[b], st));
        GX_CUDA(g, cudaStreamWaitEvent(sout, e_cmp[b], 0));
        for (int s = 0; s < g->Ns; ++s)
            GX_CUDA(g, cudaMemcpyAsync(oh + ((size_t)s * g->Nm + m0) * per_m, dout + (size_t)s * nm * per_m,
                                       (size_t)nm * per_m * sizeof(float2), cudaMemcpyDeviceToHost, sout));
        GX_CUDA(g, cudaEventRecord(e_out[b], sout));
    }
    GX_CUDA(g, cudaStreamWaitEvent(st, e_out[nb - 1], 0));
    if (use_graph) {
        cudaGraph_t graph = nullptr;
        GX_CUDA(g, cudaStreamEndCapture(st, &graph));
        cudaError_t e = cudaGraphInstantiate(&g->host_graph, graph, 0);
        cudaGraphDestroy(graph);
        if (e != cudaSuccess) return cuda_fail(g, e, "cudaGraphInstantiate");
        g->hg_g = g_host; g->hg_phi = phi_host; g->hg_out = out_host;
        GX_CUDA(g, cudaGraphLaunch(g->host_graph, st));
    }
    GX_CUDA(g, cudaStreamSynchronize(st));
    if (std::getenv("GX_HOST_TRACE") && !use_graph) {      // development aid: stage completion times of this call
        for (int b = 0; b < nb; ++b) {
            float a = 0, c = 0, d = 0;
            cudaEventElapsedTime(&a, e_start, e_in[b]);
            cudaEventElapsedTime(&c, e_start, e_cmp[b]);
            cudaEventElapsedTime(&d, e_start, e_out[b]);
            std::fprintf(stderr, "gx host pipeline: block %d in %.0f us, computed %.0f us, out %.0f us\n", b, a * 1e3, c * 1e3, d * 1e3);
        }
    }
    return GX_OK;
}

int gx_field_solve(gx_grid* g, const void* g_dev, void* phi_dev, void* cuda_stream) {
    if (!g) return GX_ERR_ARG;
    if (!g_dev || !phi_dev) return fail(g, GX_ERR_ARG, "gx_field_solve: null pointer");
    if (!g->geo_set || !g->have_lin_geo) return fail(g, GX_ERR_STATE, "gx_field_solve: full geometry not set");
    cudaError_t e = gx::lin_field_solve(g->lin, (const float2*)g_dev, (float2*)phi_dev, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(g, e, "gx_field_solve");
    return GX_OK;
}

int gx_linear_rhs(gx_grid* g, const void* g_dev, const void* phi_dev, void* out_dev, void* cuda_stream) {
    if (!g) return GX_ERR_ARG;
    if (!g_dev || !phi_dev || !out_dev) return fail(g, GX_ERR_ARG, "gx_linear_rhs: null pointer");
    if (overlap(g_dev, out_dev, (size_t)g->Ns * g->Nm * g->Nl * g->Nz * g->nk * sizeof(float2)))
        return fail(g, GX_ERR_ARG, "gx_linear_rhs: out must not alias g");
    if (misaligned(g_dev) || misaligned(phi_dev) || misaligned(out_dev))
        return fail(g, GX_ERR_ARG, "gx_linear_rhs: device pointers must be 16-byte aligned");
    if (!g->geo_set || !g->have_lin_geo) return fail(g, GX_ERR_STATE, "gx_linear_rhs: full geometry not set");
    cudaError_t e = gx::lin_rhs(g->lin, (const float2*)g_dev, (const float2*)phi_dev, (float2*)out_dev,
                                /*accumulate=*/false, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(g, e, "gx_linear_rhs");
    return GX_OK;
}

// Same kernels and launch configuration as gx_linear_rhs; the only difference is where the moments workspace lives.
// Calls no cudaMalloc / cudaFree / allocating library routine (lin_rhs only launches kernels).
int gx_linear_rhs_static(gx_grid* g, const void* g_dev, const void* phi_dev, void* out_dev, void* cuda_stream) {
    if (!g) return GX_ERR_ARG;
    if (!g_dev || !phi_dev || !out_dev) return fail(g, GX_ERR_ARG, "gx_linear_rhs_static: null pointer");
    const unsigned long long need = 3ull * (unsigned long long)g->Ns * g->Nz * (unsigned long long)g->nk;
    if (need > kStaticMomElems)
        return fail(g, GX_ERR_UNSUPPORTED, "gx_linear_rhs_static: moments workspace of " + std::to_string(need) +
                    " complex values (3 Ns Nz nakx naky) exceeds the static scratch of " + std::to_string(kStaticMomElems) +
                    " (GX_STATIC_SCRATCH_ELEMS); use gx_linear_rhs");
    if (overlap(g_dev, out_dev, (size_t)g->Ns * g->Nm * g->Nl * g->Nz * g->nk * sizeof(float2)))
        return fail(g, GX_ERR_ARG, "gx_linear_rhs_static: out must not alias g");
    if (misaligned(g_dev) || misaligned(phi_dev) || misaligned(out_dev))
        return fail(g, GX_ERR_ARG, "gx_linear_rhs_static: device pointers must be 16-byte aligned");
    if (!g->geo_set || !g->have_lin_geo) return fail(g, GX_ERR_STATE, "gx_linear_rhs_static: full geometry not set");
    if (!g->static_mom) return fail(g, GX_ERR_STATE, "gx_linear_rhs_static: static scratch address not resolved");
    gx::LinTables t = g->lin;            // plain struct of device pointers and scalars: a copy owns nothing
    t.mom = g->static_mom;               // every element read is written by lin_moments_kernel earlier in this call
    cudaError_t e = gx::lin_rhs(t, (const float2*)g_dev, (const float2*)phi_dev, (float2*)out_dev,
                                /*accumulate=*/false, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(g, e, "gx_linear_rhs_static");
    return GX_OK;
}

namespace {
// One Runge-Kutta stage st.out = a y0 + b (y + dt rhs).  Where the right-hand side ends in the separate inverse-Laguerre
// kernel, that kernel applies the stage itself (the rhs is then never stored: two passes over the state saved).
struct RkStage { const float2* y0; const float2* y; float2* out; float a, b, dt; };
int rhs_impl(gx_grid* g, const void* g_dev, void* out_dev, void* cuda_stream, const RkStage* stage, bool* folded);
}  // namespace

int gx_rhs(gx_grid* g, const void* g_dev, void* out_dev, void* cuda_stream) {
    return rhs_impl(g, g_dev, out_dev, cuda_stream, nullptr, nullptr);
}

namespace {
int rhs_impl(gx_grid* g, const void* g_dev, void* out_dev, void* cuda_stream, const RkStage* stage, bool* folded) {
    if (folded) *folded = false;
    if (!g) return GX_ERR_ARG;
    if (!g_dev || !out_dev) return fail(g, GX_ERR_ARG, "gx_rhs: null pointer");
    if (overlap(g_dev, out_dev, (size_t)g->Ns * g->Nm * g->Nl * g->Nz * g->nk * sizeof(float2)))
        return fail(g, GX_ERR_ARG, "gx_rhs: out must not alias g");
    if (misaligned(g_dev) || misaligned(out_dev)) return fail(g, GX_ERR_ARG, "gx_rhs: device pointers must be 16-byte aligned");
    if (!g->geo_set || !g->have_lin_geo) return fail(g, GX_ERR_STATE, "gx_rhs: full geometry not set");
    if (!g->ks) return fail(g, GX_ERR_UNSUPPORTED, "no kernel instantiation for this (Nx,Ny)");
    int rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if ((rc = gx_field_solve(g, g_dev, g->dphi_rhs, cuda_stream))) return rc;
    const bool concurrent = !g->ks->fused_laguerre && !g->profile && std::getenv("GX_RHS_SERIAL") == nullptr;
    if (!concurrent) {
        if ((rc = gx_nonlinear_rhs(g, g_dev, g->dphi_rhs, out_dev, cuda_stream))) return rc;
        cudaError_t e = gx::lin_rhs(g->lin, (const float2*)g_dev, g->dphi_rhs, (float2*)out_dev, /*accumulate=*/true, st);
        if (e != cudaSuccess) return cuda_fail(g, e, "gx_rhs");
        return GX_OK;
    }
    // The linear terms (memory-bound, they write out) run on a second stream under the chi and bracket kernels
    // (FP32-bound, they do not touch out); the inverse-Laguerre kernel then adds -N on top.
    if (!g->st_lin) {
        GX_CUDA(g, cudaStreamCreateWithFlags(&g->st_lin, cudaStreamNonBlocking));
        GX_CUDA(g, cudaEventCreateWithFlags(&g->ev_phi, cudaEventDisableTiming));
        GX_CUDA(g, cudaEventCreateWithFlags(&g->ev_lin, cudaEventDisableTiming));
    }
    GX_CUDA(g, cudaEventRecord(g->ev_phi, st));
    GX_CUDA(g, cudaStreamWaitEvent(g->st_lin, g->ev_phi, 0));
    cudaError_t e = gx::lin_rhs(g->lin, (const float2*)g_dev, g->dphi_rhs, (float2*)out_dev, /*accumulate=*/false, g->st_lin);
    if (e != cudaSuccess) return cuda_fail(g, e, "gx_rhs");
    GX_CUDA(g, cudaEventRecord(g->ev_lin, g->st_lin));
    NlParams p = make_params(g, g_dev, g->dphi_rhs, out_dev);
    p.accumulate = 1;
    if (stage && std::getenv("GX_RK_UNFUSED") == nullptr) {
        p.st_y0 = stage->y0; p.st_y = stage->y; p.st_out = stage->out;
        p.st_a = stage->a; p.st_b = stage->b; p.st_dt = stage->dt;
        if (folded) *folded = true;
    }
    return nl_enqueue(g, p, g->Nm, true, g->dcount, &g->calls, st, nullptr, g->ev_lin);
}
}  // namespace

int gx_ssprk3_step(gx_grid* g, void* g_dev, double dt, void* cuda_stream) {
    if (!g) return GX_ERR_ARG;
    if (!g_dev || !(dt > 0)) return fail(g, GX_ERR_ARG, "gx_ssprk3_step: null pointer or dt <= 0");
    if (!g->geo_set || !g->have_lin_geo) return fail(g, GX_ERR_STATE, "gx_ssprk3_step: full geometry not set");
    const size_t n = (size_t)g->Ns * g->Nm * g->Nl * g->Nz * g->nk;
    int rc;
    if (!g->drk_y) {
        if ((rc = dev_alloc(g, &g->drk_y, n))) return rc;
        if ((rc = dev_alloc(g, &g->drk_k, n))) return rc;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    float2* y0 = (float2*)g_dev;
    const float h = (float)dt;
    const int blocks = (int)std::min<size_t>((n + 255) / 256, 148 * 16);
    // Stage results may overwrite the state the right-hand side was evaluated on (stage 2): the inverse-Laguerre block
    // of an (s,m,z) runs after every bracket unit of that (s,m,z) has arrived and after the linear kernels (event),
    // and no other unit reads those planes.
    const RkStage stages[3] = {{y0, y0, g->drk_y, 0.f, 1.f, h},                              // g1
                               {y0, g->drk_y, g->drk_y, 0.75f, 0.25f, h},                    // g2
                               {y0, g->drk_y, y0, 1.f / 3.f, 2.f / 3.f, h}};                 // g(t+dt)
    for (int i = 0; i < 3; ++i) {
        bool folded = false;
        if ((rc = rhs_impl(g, i == 0 ? y0 : g->drk_y, g->drk_k, cuda_stream, &stages[i], &folded))) return rc;
        if (!folded)
            gx::rk_stage_kernel<<<blocks, 256, 0, st>>>(stages[i].out, stages[i].y0, stages[i].y, g->drk_k, stages[i].a, stages[i].b, h, n);
    }
    GX_CUDA(g, cudaGetLastError());
    return GX_OK;
}

int gx_query(gx_grid* g, int what, long long* value) {
    if (!g || !value) return GX_ERR_ARG;
    switch (what) {
        case GX_Q_NAKX: *value = g->nakx; break;
        case GX_Q_NAKY: *value = g->naky; break;
        case GX_Q_NJ: *value = g->J; break;
        case GX_Q_G_ELEMS: *value = (long long)g->Ns * g->Nm * g->Nl * g->Nz * g->nk; break;
        case GX_Q_PHI_ELEMS: *value = (long long)g->Nz * g->nk; break;
        case GX_Q_WORKSPACE_BYTES: *value = (long long)g->bytes; break;
        case GX_Q_LAUNCHES_PER_NL:        // a8 inside the bracket kernel (row family, J <= 5, Nl <= 4): chi + bracket
            *value = (g->ks && g->ks->launch_call) ? 1
                   : (g->ks && (g->ks->fused_laguerre || (g->ks->closer && g->J <= 5 && g->Nl <= 4 && !std::getenv("GX_A8_KERNEL")))) ? 2 : 3;
            break;
        case GX_Q_LAUNCHES_PER_RHS: *value = ((g->ks && g->ks->launch_call) ? 1 : (g->ks && g->ks->fused_laguerre) ? 2 : 3) + gx::kLinLaunchesFieldSolve + gx::kLinLaunchesRhs; break;
        case GX_Q_NL_FLOPS: *value = nl_flops(g); break;
        case GX_Q_KERNEL_FAMILY: *value = g->ks ? g->ks->family : -1; break;
        case GX_Q_NL_BYTES:
            *value = 8LL * (2LL * g->Ns * g->Nm * g->Nl * g->Nz * g->nk + (long long)g->Nz * g->nk);
            break;
        default: return fail(g, GX_ERR_ARG, "gx_query: unknown code");
    }
    return GX_OK;
}

int gx_export_maps(gx_grid* g, int* kx_index, int* ky_index, int* pad_row, unsigned char* mask,
                   double* lag_nodes, double* lag_weights) {
    if (!g) return GX_ERR_ARG;
    for (int i = 0; i < g->nakx; ++i) {
        const int a = i <= g->K ? i : i - g->nakx;
        if (kx_index) kx_index[i] = a;
        if (pad_row) pad_row[i] = a >= 0 ? a : a + g->Nx;
    }
    if (ky_index)
        for (int q = 0; q < g->naky; ++q) ky_index[q] = q;
    if (mask) {
        const int Nyc = g->Ny / 2 + 1;
        for (int r = 0; r < g->Nx; ++r)
            for (int q = 0; q < Nyc; ++q)
                mask[(size_t)r * Nyc + q] = ((r <= g->K || r >= g->Nx - g->K) && q <= g->Q) ? 1 : 0;
    }
    for (int j = 0; j < g->J; ++j) {
        if (lag_nodes) lag_nodes[j] = g->xj[j];
        if (lag_weights) lag_weights[j] = g->wj[j];
    }
    return GX_OK;
}

int gx_export_tables(gx_grid* g, float* T, float* Tinv, float* M) {
    if (!g) return GX_ERR_ARG;
    if (T) std::memcpy(T, g->hT.data(), g->hT.size() * sizeof(float));
    if (Tinv) std::memcpy(Tinv, g->hTinv.data(), g->hTinv.size() * sizeof(float));
    if (M) {
        if (!g->geo_set) return fail(g, GX_ERR_STATE, "gx_export_tables: geometry not set");
        GX_CUDA(g, cudaMemcpy(M, g->dM, (size_t)g->Ns * g->Nz * g->J * g->nk * sizeof(float), cudaMemcpyDeviceToHost));
    }
    return GX_OK;
}

const char* gx_last_error(gx_grid* g) { return g ? g->err.c_str() : "null handle"; }

}  // extern "C"
