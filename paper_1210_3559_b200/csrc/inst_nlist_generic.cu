// inst_nlist_generic.cu -- instantiations of nlist_kernel<LPA, 0, 0, FORCE, ENERGY, MIXED> (see sc_dispatch.h)
#include "sc_dispatch.h"

namespace scmd {
namespace {
template <int LPA>
cudaError_t launch(int block, const NlistArgs &a, bool force, bool energy, bool mixed, cudaStream_t st) {
    const int n_pairs = (a.n_atoms + 1) / 2;
    const int grid = (n_pairs + a.pairs_per_cta - 1) / a.pairs_per_cta;
    auto go = [&](auto kernel) -> cudaError_t {
        kernel<<<grid, block, 0, st>>>(a);
        return cudaGetLastError();
    };
    if (!mixed) {
        if (!force) return a.shift_m != 0.0 ? go(nlist_kernel<LPA, 0, 0, false, false, false, true>)
                                          : go(nlist_kernel<LPA, 0, 0, false, false, false>);
        if (energy) return go(nlist_kernel<LPA, 0, 0, true, true, false>);
        return go(nlist_kernel<LPA, 0, 0, true, false, false>);
    }
    if (!force) return a.shift_m != 0.0 ? go(nlist_kernel<LPA, 0, 0, false, false, true, true>)
                                          : go(nlist_kernel<LPA, 0, 0, false, false, true>);
    if (energy) return go(nlist_kernel<LPA, 0, 0, true, true, true>);
    return go(nlist_kernel<LPA, 0, 0, true, false, true>);
}
}  // namespace

cudaError_t launch_nlist_generic(int lpa, int block, const NlistArgs &a, bool force, bool energy, bool mixed, cudaStream_t st) {
    switch (lpa) {
        case 8: return launch<8>(block, a, force, energy, mixed, st);
        case 16: return launch<16>(block, a, force, energy, mixed, st);
        case 32: return launch<32>(block, a, force, energy, mixed, st);
    }
    return cudaErrorInvalidConfiguration;
}
}  // namespace scmd
