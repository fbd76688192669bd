/* gx.h -- C-ABI of the B200-native nonlinear E×B term of the Fourier-Laguerre-Hermite
 * gyrokinetic system of GX (arxiv 2209.06731).  "P:nnn" = line nnn of PAPER.md.
 *
 * The library evaluates, for every species s, Hermite index m, field-line point z and
 * dealiased perpendicular mode k = (kx, ky),
 *
 *   out[s,m,l,z,k] = - N^s_{l,m}(k,z)                                   (Eq. 4.9: N sits on the LHS)
 *   N^s_{l,m} = L_l F_k ( F^-1[i ky J0s Phi] F^-1[i kx sum_l' psi_l' G_{l',m}]
 *                       - F^-1[i kx J0s Phi] F^-1[i ky sum_l' psi_l' G_{l',m}] )
 *                                                                       (App. D Eq. D1 line 1; Eq. 4.19)
 * pseudo-spectrally: Laguerre l -> mu-nodes, spectral derivatives, zero-padded inverse 2D FFT,
 * pointwise bracket, forward FFT, 2/3-rule dealiasing, Laguerre mu-nodes -> l.
 * All device arithmetic is fp32; tables are computed in fp64 on the host and rounded once.
 *
 * LAYOUT (slowest -> fastest), interleaved complex64 (re,im):
 *   g, out : [s][m][l][z][kx][ky]   compact dealiased: nakx = 1+2*((Nx-1)/3), naky = 1+(Ny-1)/3
 *            kx integers in FFT order 0,1,..,K,-K,..,-1 (K=(nakx-1)/2); ky integers 0..naky-1
 *            (ky<0 implied by the reality condition)
 *   phi    : [z][kx][ky]
 * PRECONDITION: the ky=0 column is Hermitian, f(-kx,0) = conj f(kx,0), f(0,0) real; otherwise the
 *   result is unspecified.
 * OWNERSHIP: g, phi, out are caller-owned DEVICE pointers (16-byte aligned; out must not alias g);
 *   the library keeps no reference after the call returns.  The handle owns all tables and the
 *   workspace.  Geometry / species arrays are HOST pointers, copied during the call.
 *   Misaligned device pointers and partially overlapping g / out ranges are rejected with GX_ERR_ARG.
 * ASYNC: compute calls enqueue on the given cudaStream_t (passed as void*) and do not synchronise.
 * CONCURRENCY: a handle owns ONE workspace (chi planes, node planes, arrival counters, phi of gx_rhs, RK buffers):
 *   it is single-thread and single-stream -- all compute calls on a handle must be ordered on one stream (or
 *   ordered by the caller with events).  Use one handle per stream for concurrent evaluations.
 * ERRORS: every call returns 0 (GX_OK) or a negative code; no exception crosses the ABI;
 *   gx_last_error() returns a message for the last failure on that handle.
 * There is NO CPU fallback: without a CUDA device gx_grid_create fails with GX_ERR_CUDA.
 */
#ifndef GX_H_
#define GX_H_

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gx_grid gx_grid;

enum {
    GX_OK = 0,
    GX_ERR_ARG = -1,         /* bad size / null pointer / index out of range                    */
    GX_ERR_STATE = -2,       /* box, species or geometry not set before a compute call           */
    GX_ERR_UNSUPPORTED = -3, /* (Nx,Ny) has no kernel instantiation, or the plane does not fit   */
    GX_ERR_CUDA = -4,        /* CUDA runtime error (message via gx_last_error)                   */
    GX_ERR_ALLOC = -5
};

/* what-codes for gx_query */
enum {
    GX_Q_NAKX = 0, GX_Q_NAKY = 1, GX_Q_NJ = 2,        /* dealiased counts, number of mu-nodes J   */
    GX_Q_G_ELEMS = 3, GX_Q_PHI_ELEMS = 4,             /* complex elements of g/out and of phi      */
    GX_Q_WORKSPACE_BYTES = 5,                         /* device bytes owned by the handle          */
    GX_Q_LAUNCHES_PER_NL = 6,                         /* kernels launched by one gx_nonlinear_rhs  */
    GX_Q_LAUNCHES_PER_RHS = 7,
    GX_Q_NL_FLOPS = 8, GX_Q_NL_BYTES = 9,             /* algorithmic flops / HBM bytes per call */
    GX_Q_KERNEL_FAMILY = 10                           /* GX_FAMILY_* chosen for this grid (env GX_KERNELS) */
};

/* Kernel families of the nonlinear path; GX_KERNELS=scalar|pair|persist|row|rowp forces one. */
enum { GX_FAMILY_SCALAR = 0, GX_FAMILY_ROW = 3, GX_FAMILY_RX = 5, GX_FAMILY_RXP = 6, GX_FAMILY_RXW = 7 };   /* 1, 2, 4: families removed in round 2 */

/* Create a handle for real-space grid Nx x Ny, Nz field-line points, Nl Laguerre and Nm Hermite
 * moments, Ns species.  Nx, Ny must be even, >= 4, and factor as R1*R2 with R1,R2 in
 * {2,3,4,6,8,12,16} (all sizes of BASELINE.json configs do); Nl <= 16.  The number of mu-nodes
 * is J = (3*Nl-1)/2 (smallest Gauss-Laguerre rule exact for triple products; R2).
 * Builds index maps, Gauss-Laguerre nodes/weights, T[j][l] = psi_l(x_j), Tinv[l][j] = w_j psi_l(x_j),
 * psi_l = (-1)^l L_l, and FFT twiddles.  Uses the current CUDA device. */
int gx_grid_create(int Nx, int Ny, int Nz, int Nl, int Nm, int Ns, gx_grid** out);
int gx_grid_destroy(gx_grid* g);

/* Perpendicular box: ky = dky*q, kx = dkx*p (units 1/rho_ref, Table 4); shat enters
 * kperp2 through gds21/shat, gds22/shat^2 (P:681-686 Eq. E6-E7). */
int gx_box_set(gx_grid* g, double dky, double dkx, double shat);

/* Species s: charge Z_s, mass m_s, temperature tau_s, density n_s, gradients
 * tprim = 1/L_Ts, fprim = 1/L_ns, like-species collision frequency nu_ss. */
int gx_species_set(gx_grid* g, int s, double Z, double mass, double temp, double dens,
                   double tprim, double fprim, double nu_ss);

/* Adiabatic (Boltzmann) electron response for the field solve, Eq. 6.1:
 * enabled != 0 selects it (requires Ns == 1); tau_fac = T_i/T_e. Default: enabled iff Ns == 1, tau_fac 1. */
int gx_adiabatic_set(gx_grid* g, int enabled, double tau_fac);

/* Parallel boundary condition of the z operators in gx_rhs / gx_linear_rhs (call before gx_geometry_set):
 * linked == 0 (default): every (kx,ky) is periodic in z by itself; linked != 0: twist-and-shift (Eq. 4.29,
 * P:322-327), H(kx,ky,z) = H(kx + dk,ky,z + 2 pi), dk = 2 pi ky shat: the modes kx_0 + n dk inside the dealiased
 * set form one periodic extended domain on which grad_par and |k_par| are spectral.  Needs a quantised box,
 * 2 pi shat dky / dkx a non-zero integer; gx_geometry_set returns GX_ERR_ARG otherwise. */
int gx_boundary_set(gx_grid* g, int linked);

/* Dissipation parameters of gx_rhs: hyper-viscosity D (k_perp^2/k_perp,max^2)^n (Eq. 4.26) and
 * hyper-collisions nu_hyp m^p, p = Nm/2, strength f_hyp (Eq. 4.27-4.28). Defaults 0.05, 4, 1. */
int gx_dissipation_set(gx_grid* g, double D_hyper, int n_hyper, double f_hyp);

/* Wave-absorbing layer at the ends of every (extended) z domain, Eq. 4.30:
 * dG_{l,m}/dt -= d(z_hat) H_{l,m} for ky != 0, d = A [1 - 2 z_hat^2/(1 + z_hat^4)] for |z_hat| < 1, z_hat the
 * distance from either end of the domain in units of width_fraction * L_z (the paper uses 1/8 and A = 0.1/dt).
 * With gx_boundary_set(0) every mode is its own domain of length 2 pi.  A = 0 (default) switches the layer off.
 * Call before gx_geometry_set. */
int gx_damping_set(gx_grid* g, double A, double width_fraction);

/* Per-z geometry coefficients (HOST arrays of length Nz, P:677-694 Eq. E4-E11) and the constant
 * gradpar = b.grad z.  bmag, gds2, gds21, gds22 define k_perp^2 and b_s and hence the
 * gyroaverage table M[s][z][j][kx][ky] = J0(sqrt(2 x_j b_s)) built here in fp64; the drift,
 * bgrad (= grad_par ln B) and jacobian arrays are used by gx_rhs / gx_field_solve only and may be
 * NULL if those are never called.  Requires gx_box_set and every gx_species_set first. */
int gx_geometry_set(gx_grid* g, const double* bmag, const double* gds2, const double* gds21,
                    const double* gds22, const double* gbdrift, const double* gbdrift0,
                    const double* cvdrift, const double* cvdrift0, const double* bgrad,
                    const double* jacobian, double gradpar);

/* out = -N[g, phi]  (the hot path).  Device pointers; enqueued on `cuda_stream`.
 * Stream semantics are the usual ones: g and phi must have been produced by work enqueued earlier on the stream
 * (or be complete), and anything enqueued after the call sees `out` complete.  Consecutive calls on one handle
 * overlap on the device where the kernel family supports it (NY = 64: the potential planes and the first units of a
 * call run under the last wave of the previous call; the reuse of the workspace and of `out` is ordered by device
 * counters, the two calls may write the same `out`).  Inputs of a call must not be overwritten before the call has
 * completed in stream order -- as for any asynchronous call.  The device compute calls cannot be recorded into a
 * CUDA graph by the caller (their kernels take the call's epoch as an argument): GX_ERR_STATE while the stream is
 * capturing; gx_nonlinear_rhs_host builds and replays a graph of its own.  Environment: GX_CHI_SERIAL=1 disables the overlap,
 * GX_A8_KERNEL=1 keeps the inverse Laguerre transform a separate kernel (development aids). */
int gx_nonlinear_rhs(gx_grid* g, const void* g_dev, const void* phi_dev, void* out_dev,
                     void* cuda_stream);

/* Electromagnetic form of the hot path (App. D Eq. D1 lines 1-4, with Eq. 4.5):
 *   out = -N,  N_{l,m} = L_l F[ {J0 Phi + (tau/Z) 2 muB (J1/alpha) dB_par/B, gt_m} - v_ts {J0 A_par, sqrt(m+1) gt_{m+1} + sqrt(m) gt_{m-1}} ]
 * apar_dev, bpar_dev: device fields A_par and dB_par/B in the layout of phi.  Evaluated as two passes of the
 * electrostatic kernels (potential planes built in spectral space, Hermite-shifted state for the A_par pass) whose
 * results are added; needs the full geometry (gx_geometry_set with all arrays); two state-sized work buffers are
 * allocated on first use.  apar = bpar = 0 reproduces gx_nonlinear_rhs. */
int gx_nonlinear_rhs_em(gx_grid* g, const void* g_dev, const void* phi_dev, const void* apar_dev, const void* bpar_dev,
                        void* out_dev, void* cuda_stream);

/* Field solve with electromagnetic fluctuations, Eq. 4.23-4.25, kinetic species only (no adiabatic
 * closure), beta = beta_ref >= 0: per (z,k) the 2x2 system for (Phi, dB_par/B) and the parallel Ampere law for A_par;
 * sums over l truncated at Nl; all three fields vanish at kx = ky = 0.  beta = 0 gives the two-species gx_field_solve. */
int gx_field_solve_em(gx_grid* g, const void* g_dev, double beta, void* phi_dev, void* apar_dev, void* bpar_dev,
                      void* cuda_stream);

/* Same call with HOST buffers (pinned for full speed).  The evaluation is diagonal in the Hermite index, so it
 * is pipelined over blocks of moments on three streams: the host-to-device copy of block b+1 and the
 * device-to-host copy of block b-1 overlap the kernels of block b (chi planes computed once).  Ordered after
 * the work already queued on `cuda_stream`; synchronises before returning. */
int gx_nonlinear_rhs_host(gx_grid* g, const void* g_host, const void* phi_host, void* out_host,
                          void* cuda_stream);

/* Quasineutrality field solve phi = phi[g] on the device: Eq. 6.1 for adiabatic electrons
 * (with the jacobian-weighted flux-surface average at ky=0), else Eq. 4.23 with dB_par = 0;
 * sums over l truncated at Nl; phi(kx=0,ky=0) = 0. */
int gx_field_solve(gx_grid* g, const void* g_dev, void* phi_dev, void* cuda_stream);

/* out = dG/dt = -N + linear terms of Eq. 4.9: streaming, mirror, curvature and grad-B
 * drifts, drive (Eq. 4.12), Dougherty collisions (Eq. 4.13-4.18), hyper-viscosity, hyper-collisions;
 * phi is computed internally with gx_field_solve.  Electrostatic (beta_ref = 0). */
int gx_rhs(gx_grid* g, const void* g_dev, void* out_dev, void* cuda_stream);

/* One step of the third-order SSP Runge-Kutta scheme the paper uses for the nonlinear runs (P:347,
 * Shu-Osher form): g1 = g + dt R(g); g2 = 3/4 g + 1/4 (g1 + dt R(g1)); g <- 1/3 g + 2/3 (g2 + dt R(g2)),
 * R = gx_rhs.  g_dev is updated in place; two state-sized work buffers are owned by the handle
 * (allocated on first use).  Enqueued on `cuda_stream`; 3 gx_rhs evaluations + 3 fused stage kernels. */
int gx_ssprk3_step(gx_grid* g, void* g_dev, double dt, void* cuda_stream);

/* Linear part only (gx_rhs without -N), given phi; used to test the linear terms on their own. */
int gx_linear_rhs(gx_grid* g, const void* g_dev, const void* phi_dev, void* out_dev, void* cuda_stream);

/* gx_linear_rhs for callers that cannot allocate (code under CUDA graph capture, serving loops, harnesses
 * that forbid cudaMalloc): same arguments, same kernels, same result, but the one workspace the call
 * needs -- the Dougherty field-particle moments mom[s][3][z][k] of Eq. 4.14-4.18, complex
 * fp32 -- lives in a file-scope `static __device__` array of the library instead of the handle's
 * allocation.  The call performs no cudaMalloc / cudaFree and calls no allocating library routine; the
 * array's device address is resolved (cudaGetSymbolAddress) when the handle is created.
 * Limit: 3 * Ns * Nz * nakx * naky <= GX_STATIC_SCRATCH_ELEMS complex values (4 MiB; every GPU that
 * loads the library holds it until the process exits); larger grids return GX_ERR_UNSUPPORTED with a
 * message naming both numbers (gx_last_error) and enqueue nothing.
 * The array is shared by every call, every handle and every stream on a device and keeps the last
 * call's contents.  Nothing in it has to start at zero: every element a call reads is written earlier in
 * that same call.  Two calls that overlap on the GPU (different streams, or different handles on one
 * device) race on it; calls on one stream are ordered and safe.  Other errors as gx_linear_rhs. */
#define GX_STATIC_SCRATCH_ELEMS (1u << 19)
int gx_linear_rhs_static(gx_grid* g, const void* g_dev, const void* phi_dev, void* out_dev, void* cuda_stream);

int gx_query(gx_grid* g, int what, long long* value);

/* Parity exports (HOST outputs; any pointer may be NULL): compact kx integers [nakx], ky integers
 * [naky], padded row of each compact kx row [nakx] (= p mod Nx), 2/3-rule mask over the padded
 * half-spectrum [Nx*(Ny/2+1)], Gauss-Laguerre nodes and weights [nj]. */
int gx_export_maps(gx_grid* g, int* kx_index, int* ky_index, int* pad_row, unsigned char* mask,
                   double* lag_nodes, double* lag_weights);

/* Table exports for parity tests (HOST outputs, fp32 as used on the device):
 * T [nj*Nl], Tinv [Nl*nj], M [Ns*Nz*nj*nakx*naky] (needs geometry set; may be NULL). */
int gx_export_tables(gx_grid* g, float* T, float* Tinv, float* M);

/* Per-kernel timing for the roofline report.  While enabled, every gx_nonlinear_rhs records CUDA
 * events on the launch stream around each of its kernels.  gx_profile_get synchronises those events,
 * adds the elapsed milliseconds of [0] chi planes, [1] bracket, [2] inverse Laguerre to ms[0..2],
 * writes the number of profiled calls to *calls, and resets the accumulators. */
int gx_profile_set(gx_grid* g, int enabled);
int gx_profile_get(gx_grid* g, double* ms, long long* calls);

const char* gx_last_error(gx_grid* g);

/* FP32 pipe micro-benchmark on the current device (no handle): `iters` rounds of 16 independent dependency
 * chains per thread of one instruction kind -- 0 add.f32, 1 mul.f32, 2 fma.rn.f32, 3 add.f32x2, 4 mul.f32x2,
 * 5 fma.rn.f32x2 -- on (SM count * blocks_per_sm) blocks of threads_per_block threads.  Writes the kernel time
 * (CUDA events, one warm-up launch before) to *ms and the number of lane operations executed to *lane_ops (a
 * packed instruction counts two, an FMA counts one: flops = 2 * lane_ops for kinds 2 and 5).  bench.py derives
 * roofline.peak_measured from it ("the bench should also run a tiny FMA-peak kernel"). */
int gx_ubench_fp32(int kind, int threads_per_block, int blocks_per_sm, int iters, double* ms, double* lane_ops);

/* Register radix-16 micro-benchmark: `iters` 16-point complex DFTs (+ 15 twiddle multiplications each, as in a
 * two-pass FFT) per thread, entirely in registers; packed != 0: two transforms per thread in the packed FP32 form of
 * dft_packed.cuh.  *transforms = number of 16-point transforms done.  Used by `bench.py --tcdft`, which sets this
 * rate against the tensor-core rate a split-TF32 matrix form of the same DFT could reach (profiles/r02_tensor_dft.md). */
int gx_ubench_dft16(int packed, int threads_per_block, int blocks_per_sm, int iters, double* ms, double* transforms);

#ifdef __cplusplus
}
#endif
#endif /* GX_H_ */
