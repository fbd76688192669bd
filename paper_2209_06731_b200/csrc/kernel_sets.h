// kernel_sets.h -- launcher tables of the kernel families; one translation unit per family (parallel build).
#pragma once
#include <cuda_runtime.h>

#include <algorithm>

#include "../../include/gx.h"
#include "nl_kernels.cuh"

namespace gxhost {
using gx::NlParams;

// per-(Nx,Ny) kernel launchers of one family
struct KernelSet {
    int Nx, Ny;
    int smem_bytes;
    int family;          // GX_FAMILY_* of include/gx.h
    cudaError_t (*prepare)();                    // opt-in shared-memory attributes, on the current device (gx_grid_create)
    cudaError_t (*launch_chi)(const NlParams&, int units, cudaStream_t);
    cudaError_t (*launch_bracket)(const NlParams&, int units, cudaStream_t);
    bool fused_laguerre;   // the bracket kernel writes `out` itself (a8 fused): no third launch
    // one persistent kernel for the whole call (chi planes + bracket units + a8); launch_chi/bracket unused then
    cudaError_t (*launch_call)(const NlParams&, unsigned* chi_flag, unsigned epoch, int n_items, cudaStream_t);
    // the bracket kernel can do a8 itself in the CTA that completes an (s,m,z) (NlParams::a8_target != 0)
    bool closer = false;
    // chi launcher with the PDL attribute: the chi planes of call N+1 start under the tail of call N (other dchi buffer)
    // (bracket-sized CTAs: they fit next to the bracket CTAs of the previous call's last wave)
    cudaError_t (*launch_chi_pdl)(const NlParams&, int units, cudaStream_t) = nullptr;
    cudaError_t (*launch_chi_pdl_wide)(const NlParams&, int units, cudaStream_t) = nullptr;   // same, launch_chi's CTA shape
    // the kernels work on the transposed plane (RowCfg<..., TR = true>): the host swaps dkx / dky and the x / y twiddle
    // tables and flips the sign of the bracket
    bool transposed = false;
};

// Launch with the programmatic-stream-serialization attribute (PDL): the grid may begin before the
// previous kernel in the stream has finished; the kernel itself waits (griddepcontrol.wait) before it
// reads that kernel's output.
template <class... Args, class... Act>
cudaError_t launch_pdl(void (*kernel)(Args...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Act... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, args...);
}
template <class K> cudaError_t set_smem(K kernel, int bytes) {
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
}
inline int sm_count() {
    int dev = 0, n = 0;
    cudaGetDevice(&dev);
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
    return n;
}


const KernelSet* find_scalar(int Nx, int Ny);      // sets_scalar.cu (falls through to sets_scalar2.cu)
const KernelSet* find_scalar_more(int Nx, int Ny); // sets_scalar2.cu
const KernelSet* find_row(int Nx, int Ny);         // sets_row.cu
const KernelSet* find_rx(int Nx, int Ny, int family);   // sets_rx.cu: GX_FAMILY_RX / RXP / RXW

template <int N> const KernelSet* find_in(const KernelSet (&sets)[N], int Nx, int Ny) {
    for (const auto& k : sets)
        if (k.Nx == Nx && k.Ny == Ny) return &k;
    return nullptr;
}
}  // namespace gxhost
