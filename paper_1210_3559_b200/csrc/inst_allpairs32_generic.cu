// inst_allpairs32_generic.cu -- instantiations of allpairs32_kernel<IT, TPR, 0, 0, FORCE, ENERGY> (see sc_dispatch.h)
#include "sc_dispatch.h"

namespace scmd {
namespace {
template <int IT, int TPR>
const void *pick(bool force, bool energy) {
    if (!force) return reinterpret_cast<const void *>(allpairs32_kernel<IT, TPR, 0, 0, false, false>);
    if (energy) return reinterpret_cast<const void *>(allpairs32_kernel<IT, TPR, 0, 0, true, true>);
    return reinterpret_cast<const void *>(allpairs32_kernel<IT, TPR, 0, 0, true, false>);
}
}  // namespace

const void *allpairs32_fn_generic(int it, int tpr, bool force, bool energy) {
#define SC_CASE(IT, TPR) \
    if (it == IT && tpr == TPR) return pick<IT, TPR>(force, energy);
    SC_CASE(1, 1) SC_CASE(1, 2) SC_CASE(1, 4) SC_CASE(1, 8) SC_CASE(1, 16) SC_CASE(1, 32)
    SC_CASE(2, 1) SC_CASE(2, 2) SC_CASE(2, 4) SC_CASE(2, 8) SC_CASE(2, 16) SC_CASE(2, 32)
#undef SC_CASE
    return nullptr;
}
}  // namespace scmd
