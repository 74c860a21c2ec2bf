// inst_nlist_96.cu -- instantiations of nlist_kernel<9, 6, FORCE, ENERGY, MIXED, SHIFT> (see sc_dispatch.h)
#include "sc_dispatch.h"

namespace scmd {
cudaError_t launch_nlist_96(int grid, int block, const NlistArgs &a, bool force, bool energy, bool mixed, cudaStream_t st) {
    const size_t smem = kListRuns ? size_t(block / 32) * size_t(a.idx_cap) * sizeof(int) : 0;   // the warps' expanded rows
    auto go = [&](auto kernel) -> cudaError_t {
        if (smem > 48 * 1024) {
            cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem));
            if (e != cudaSuccess) return e;
        }
        // run-length rows: 6 resident CTAs x ~22 KB of expanded rows need the large shared-memory carve-out; index rows use
        // no shared memory and want all of it as L1 (the gathers of neighbouring rows hit the same lines)
        cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout,
                             kListRuns ? 60 : int(cudaSharedmemCarveoutMaxL1));   // 60 % of 228 KB = 6 x 22.5 KB
        kernel<<<grid, block, smem, st>>>(a);
        return cudaGetLastError();
    };
    if (!mixed) {
        if (!force) return a.shift_m != 0.0 ? go(nlist_kernel<9, 6, false, false, false, true>)
                                          : go(nlist_kernel<9, 6, false, false, false>);
        if (energy) return go(nlist_kernel<9, 6, true, true, false>);
        return go(nlist_kernel<9, 6, true, false, false>);
    }
    if (!force) return a.shift_m != 0.0 ? go(nlist_kernel<9, 6, false, false, true, true>)
                                      : go(nlist_kernel<9, 6, false, false, true>);
    if (energy) return go(nlist_kernel<9, 6, true, true, true>);
    return go(nlist_kernel<9, 6, true, false, true>);
}
}  // namespace scmd
