// sets_row.cu -- instantiations and launchers of the row family (nl_row_kernels.cuh).
#include "kernel_sets.h"
#include "nl_row_kernels.cuh"

namespace gxhost {
namespace {
// ---- row family (nl_row_kernels.cuh): whole y direction of an x row in one thread's registers; NY = 64
template <class CB, class CC> cudaError_t prepare_row() {
    cudaError_t e = set_smem(gx::chi_planes_row_kernel<CC>, CC::SMEM_BYTES);
    if (e == cudaSuccess) e = set_smem(gx::chi_planes_row_kernel<CB>, CB::SMEM_BYTES);
    if (e == cudaSuccess) e = set_smem(gx::bracket_row_kernel<CB, 1>, CB::SMEM_BYTES);
    if (e == cudaSuccess) e = set_smem(gx::bracket_row_kernel<CB, 2>, CB::SMEM_BYTES);
    return e != cudaSuccess ? e : set_smem(gx::bracket_row_kernel<CB, 0>, CB::SMEM_BYTES);
}
template <class C> cudaError_t launch_chi_row_t(const NlParams& p, int units, cudaStream_t st) {
    gx::chi_planes_row_kernel<C><<<units, C::NT, C::SMEM_BYTES, st>>>(p);
    return cudaGetLastError();
}
template <class C> cudaError_t launch_chi_row_pdl_t(const NlParams& p, int units, cudaStream_t st) {
    return launch_pdl(gx::chi_planes_row_kernel<C>, dim3(units), dim3(C::NT), C::SMEM_BYTES, st, p);
}
template <class C> cudaError_t launch_bracket_row_t(const NlParams& p, int units, cudaStream_t st) {
    const bool chain = p.done != nullptr || p.a8_target != 0u;
    if (chain && p.cluster) {       // the J node units of an (s,m,z) as one cluster, PDL attribute as for the others
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(units); cfg.blockDim = dim3(C::NT); cfg.dynamicSmemBytes = C::SMEM_BYTES; cfg.stream = st;
        cudaLaunchAttribute at[2];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        at[1].id = cudaLaunchAttributeClusterDimension;
        at[1].val.clusterDim.x = (unsigned)p.J; at[1].val.clusterDim.y = 1; at[1].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 2;
        return cudaLaunchKernelEx(&cfg, gx::bracket_row_kernel<C, 2>, p);
    }
    return chain ? launch_pdl(gx::bracket_row_kernel<C, 1>, dim3(units), dim3(C::NT), C::SMEM_BYTES, st, p)
                 : launch_pdl(gx::bracket_row_kernel<C, 0>, dim3(units), dim3(C::NT), C::SMEM_BYTES, st, p);
}
template <class CB, class CC> constexpr KernelSet make_row_set() {
    static_assert(CB::NX == CC::NX && CB::NY == CC::NY && CB::RX1 == CC::RX1 && CB::TR == CC::TR,
                  "chi and bracket kernels must share the x radices (same permuted x order)");
    return KernelSet{CB::TR ? CB::NY : CB::NX, CB::TR ? CB::NX : CB::NY, CB::SMEM_BYTES, GX_FAMILY_ROW, &prepare_row<CB, CC>,
                     &launch_chi_row_t<CC>, &launch_bracket_row_t<CB>, false, nullptr, true, &launch_chi_row_pdl_t<CB>,
                     &launch_chi_row_pdl_t<CC>, CB::TR};
}
using R96x64   = gx::RowCfg<96, 64, 8, 12, 96, 4>;
using R64x64   = gx::RowCfg<64, 64, 8, 8, 64, 6>;
using R128x64  = gx::RowCfg<128, 64, 16, 8, 128, 3>;
using R192x64  = gx::RowCfg<192, 64, 16, 12, 192, 2>;
using RC192x64 = gx::RowCfg<192, 64, 16, 12, 384, 1>;   // chi planes: < 1 wave, more threads for the x passes
using R256x64  = gx::RowCfg<256, 64, 16, 16, 256, 1>;
// physical 64 x 192 (the paper's W7-X grid) on the transposed 192 x 64 kernels
using T64x192  = gx::RowCfg<192, 64, 16, 12, 192, 2, true>;
using TC64x192 = gx::RowCfg<192, 64, 16, 12, 384, 1, true>;
using T64x96   = gx::RowCfg<96, 64, 8, 12, 96, 4, true>;
using T64x256  = gx::RowCfg<256, 64, 16, 16, 256, 1, true>;
const KernelSet kRowSets[] = {
    make_row_set<R64x64, R64x64>(), make_row_set<R128x64, R128x64>(), make_row_set<R192x64, RC192x64>(),
    make_row_set<R256x64, R256x64>(), make_row_set<T64x192, TC64x192>(), make_row_set<R96x64, R96x64>(),
    make_row_set<T64x96, T64x96>(), make_row_set<T64x256, T64x256>(),
};

}  // namespace
const KernelSet* find_row(int Nx, int Ny) { return find_in(kRowSets, Nx, Ny); }
}  // namespace gxhost

#ifdef GX_PHASE_TIMING
extern "C" int gx_debug_cta_log(long long* out) {
    return cudaMemcpyFromSymbol(out, gx::gx_cta_log, sizeof(long long) * 4 * 8192 * 16) == cudaSuccess ? 0 : -1;
}
extern "C" int gx_debug_chi_log(long long* out) {
    return cudaMemcpyFromSymbol(out, gx::gx_chi_log, sizeof(long long) * 4 * 256 * 4) == cudaSuccess ? 0 : -1;
}
extern "C" int gx_debug_phase_clocks(long long* out) {
    return cudaMemcpyFromSymbol(out, gx::gx_phase_clk, sizeof(long long) * 64 * 32) == cudaSuccess ? 0 : -1;
}
#endif
