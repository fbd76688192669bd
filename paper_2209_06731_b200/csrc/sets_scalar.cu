// sets_scalar.cu -- instantiations and launchers of the scalar family (nl_kernels.cuh).
#include "kernel_sets.h"

namespace gxhost {
namespace {
// ---- scalar family (nl_kernels.cuh): any plane with an instantiation
template <class CB, class CC> cudaError_t prepare_scalar() {
    cudaError_t e = set_smem(gx::chi_planes_kernel<CC>, CC::SMEM_BYTES);
    return e != cudaSuccess ? e : set_smem(gx::bracket_kernel<CB>, CB::SMEM_BYTES);
}
template <class C> cudaError_t launch_chi_t(const NlParams& p, int units, cudaStream_t st) {
    gx::chi_planes_kernel<C><<<units, C::NT, C::SMEM_BYTES, st>>>(p);
    return cudaGetLastError();
}
template <class C> cudaError_t launch_bracket_t(const NlParams& p, int units, cudaStream_t st) {
    return launch_pdl(gx::bracket_kernel<C>, dim3(units), dim3(C::NT), C::SMEM_BYTES, st, p);
}
template <class CB, class CC> constexpr KernelSet make_set() {
    static_assert(CB::NX == CC::NX && CB::NY == CC::NY && CB::RX1 == CC::RX1 && CB::RY1 == CC::RY1,
                  "chi and bracket kernels must share the transform radices (same permuted real-space order)");
    return KernelSet{CB::NX, CB::NY, CB::SMEM_BYTES, GX_FAMILY_SCALAR, &prepare_scalar<CB, CC>, &launch_chi_t<CC>,
                     &launch_bracket_t<CB>, false, nullptr};
}
//                  NX   NY  RX1 RX2 RY1 RY2  RB   NT MINB STAGE     (B = bracket kernel, C = chi kernel)
using B16x16   = gx::PlaneCfg<16, 16, 4, 4, 4, 4, 16, 64, 1, true>;
using B64x64   = gx::PlaneCfg<64, 64, 8, 8, 8, 8, 64, 256, 2, true>;
using B128x64  = gx::PlaneCfg<128, 64, 16, 8, 8, 8, 64, 448, 2, true>;
using C128x64  = gx::PlaneCfg<128, 64, 16, 8, 8, 8, 64, 512, 1, true>;
using B192x64  = gx::PlaneCfg<192, 64, 16, 12, 8, 8, 64, 448, 2, true>;
using C192x64  = gx::PlaneCfg<192, 64, 16, 12, 8, 8, 64, 512, 1, true>;
using B256x64  = gx::PlaneCfg<256, 64, 16, 16, 8, 8, 64, 256, 1, true>;
using B256x96  = gx::PlaneCfg<256, 96, 16, 16, 8, 12, 128, 512, 1, true>;    // RB 128: every y phase has 448-1536 items for 512 threads (RB 64 / 384 threads: 224-256 items in the two heavy phases)
using B192x192 = gx::PlaneCfg<192, 192, 16, 12, 12, 16, 16, 384, 1, false>;
using B64x192  = gx::PlaneCfg<64, 192, 8, 8, 12, 16, 16, 256, 2, true>;   // RB 16: 92 KB, two CTAs per SM
const KernelSet kKernelSets[] = {
    make_set<B16x16, B16x16>(),   make_set<B64x64, B64x64>(),     make_set<B128x64, C128x64>(),
    make_set<B192x64, C192x64>(), make_set<B256x64, B256x64>(),   make_set<B256x96, B256x96>(),
    make_set<B192x192, B192x192>(), make_set<B64x192, B64x192>(),
};

}  // namespace
const KernelSet* find_scalar(int Nx, int Ny) {
    const KernelSet* k = find_in(kKernelSets, Nx, Ny);
    return k ? k : find_scalar_more(Nx, Ny);
}
}  // namespace gxhost
