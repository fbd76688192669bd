// sets_rx.cu -- instantiations and launchers of the rx / rxp / rxw families (nl_rx_kernels.cuh).
#include "kernel_sets.h"
#include "nl_rx_kernels.cuh"

namespace gxhost {
namespace {
// ---- rx family (nl_rx_kernels.cuh): packed-FP32 x passes, row y direction, fused inverse Laguerre; NY = 64
template <class C> cudaError_t prepare_rx() {
    cudaError_t e = set_smem(gx::chi_planes_rx_kernel<C>, C::SMEM_BYTES);
    return e != cudaSuccess ? e : set_smem(gx::bracket_rx_kernel<C>, C::SMEM_BYTES);
}
template <class C> cudaError_t launch_chi_rx_t(const NlParams& p, int units, cudaStream_t st) {
    gx::chi_planes_rx_kernel<C><<<units, C::NT, C::SMEM_BYTES, st>>>(p);
    return cudaGetLastError();
}
template <class C> cudaError_t launch_bracket_rx_t(const NlParams& p, int units, cudaStream_t st) {
    return launch_pdl(gx::bracket_rx_kernel<C>, dim3(units), dim3(C::NT), C::SMEM_BYTES, st, p);
}
template <class C> constexpr KernelSet make_rx_set() {
    return KernelSet{C::NX, C::NY, C::SMEM_BYTES, GX_FAMILY_RX, &prepare_rx<C>, &launch_chi_rx_t<C>, &launch_bracket_rx_t<C>,
                     true, nullptr};
}
// ---- rxp: the rx phases in one persistent kernel, two 6-warp groups per SM
template <class C> constexpr int rxp_smem() { return 2 * C::STAGE_BYTES + C::NX * 8 + 2 * 16 * 23 * 4; }
template <class C> cudaError_t prepare_rxp() { return set_smem(gx::nl_rx_persist_kernel<C>, rxp_smem<C>()); }
template <class C> cudaError_t launch_rxp_t(const NlParams& p, unsigned* chi_flag, unsigned epoch, int n_items, cudaStream_t st) {
    static_assert(rxp_smem<C>() <= 232448, "two plane buffers do not fit in shared memory");
    const int grid = std::min(sm_count(), (n_items + 1) / 2);
    gx::nl_rx_persist_kernel<C><<<grid, 2 * C::NT, rxp_smem<C>(), st>>>(p, chi_flag, epoch);
    return cudaGetLastError();
}
template <class C> constexpr KernelSet make_rxp_set() {
    return KernelSet{C::NX, C::NY, rxp_smem<C>(), GX_FAMILY_RXP, &prepare_rxp<C>, nullptr, nullptr, true, &launch_rxp_t<C>};
}
// ---- rxw: warp-specialised pipeline (row warps + x warps), one persistent kernel
template <class C> cudaError_t prepare_rxw() { return set_smem(gx::nl_rx_pipeline_kernel<C>, gx::RxwLayout<C>::SMEM); }
template <class C> cudaError_t launch_rxw_t(const NlParams& p, unsigned* chi_flag, unsigned epoch, int n_items, cudaStream_t st) {
    using L = gx::RxwLayout<C>;
    const int grid = std::min(sm_count(), n_items);
    gx::nl_rx_pipeline_kernel<C><<<grid, L::NTHREADS, L::SMEM, st>>>(p, chi_flag, epoch);
    return cudaGetLastError();
}
template <class C> constexpr KernelSet make_rxw_set() {
    return KernelSet{C::NX, C::NY, gx::RxwLayout<C>::SMEM, GX_FAMILY_RXW, &prepare_rxw<C>, nullptr, nullptr, true, &launch_rxw_t<C>};
}

using X64x64   = gx::RxCfg<64, 64, 8, 8, 64, 6>;
using X128x64  = gx::RxCfg<128, 64, 8, 16, 128, 3>;
using X192x64  = gx::RxCfg<192, 64, 12, 16, 192, 2>;
using X256x64  = gx::RxCfg<256, 64, 16, 16, 256, 1>;
const KernelSet kRxSets[] = {make_rx_set<X64x64>(), make_rx_set<X128x64>(), make_rx_set<X192x64>(), make_rx_set<X256x64>()};
const KernelSet kRxpSets[] = {make_rxp_set<X64x64>(), make_rxp_set<X128x64>(), make_rxp_set<X192x64>()};
const KernelSet kRxwSets[] = {make_rxw_set<X64x64>(), make_rxw_set<X128x64>(), make_rxw_set<X192x64>()};

}  // namespace
const KernelSet* find_rx(int Nx, int Ny, int family) {
    if (family == GX_FAMILY_RXW) return find_in(kRxwSets, Nx, Ny);
    if (family == GX_FAMILY_RXP) return find_in(kRxpSets, Nx, Ny);
    return find_in(kRxSets, Nx, Ny);
}
}  // namespace gxhost

#ifdef GX_PHASE_TIMING
extern "C" int gx_debug_phase_clocks_rx(long long* out) {
    return cudaMemcpyFromSymbol(out, gx::gx_phase_clk, sizeof(long long) * 64 * 32) == cudaSuccess ? 0 : -1;
}
extern "C" int gx_debug_phase2_clocks(long long* out) {
    return cudaMemcpyFromSymbol(out, gx::gx_phase2_clk, sizeof(long long) * 512 * 8 * 12) == cudaSuccess ? 0 : -1;
}
#endif
