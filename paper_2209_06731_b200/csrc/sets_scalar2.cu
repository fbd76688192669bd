// sets_scalar2.cu -- further plane shapes of the scalar family (a translation unit of its own: parallel build).
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
//                  NX   NY  RX1 RX2 RY1 RY2  RB   NT MINB STAGE
using B48x48   = gx::PlaneCfg<48, 48, 6, 8, 6, 8, 16, 128, 4, true>;
using B96x96   = gx::PlaneCfg<96, 96, 8, 12, 8, 12, 32, 384, 2, true>;
using B128x96  = gx::PlaneCfg<128, 96, 16, 8, 8, 12, 32, 384, 2, true>;
using B192x96  = gx::PlaneCfg<192, 96, 16, 12, 8, 12, 32, 384, 1, true>;
using B96x192  = gx::PlaneCfg<96, 192, 8, 12, 12, 16, 16, 256, 1, true>;
const KernelSet kMoreSets[] = {
    make_set<B48x48, B48x48>(), make_set<B96x96, B96x96>(), make_set<B128x96, B128x96>(), make_set<B192x96, B192x96>(),
    make_set<B96x192, B96x192>(),
};

}  // namespace
const KernelSet* find_scalar_more(int Nx, int Ny) { return find_in(kMoreSets, Nx, Ny); }
}  // namespace gxhost
