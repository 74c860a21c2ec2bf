// sc_dispatch.h -- kernel selection across translation units.  The template instantiations of the
// sweeps live in inst_*.cu (one file per precision x exponent class so that they compile in
// parallel); scmd.cu picks a kernel through these functions.
#pragma once
#include <cuda_runtime.h>

#include "sc_allpairs.cuh"
#include "sc_cutoff.cuh"

namespace scmd {

// all-pairs sweep kernels: IT rows per thread, TPR lanes per row; nullptr if not instantiated.
// *_96: exponents (9, 6) compiled in; *_generic: exponents read from the arguments.
const void *allpairs64_fn_96(int it, int tpr, bool force, bool energy);
const void *allpairs64_fn_generic(int it, int tpr, bool force, bool energy);
const void *allpairs32_fn_96(int it, int tpr, bool force, bool energy);
const void *allpairs32_fn_generic(int it, int tpr, bool force, bool energy);

// list-driven sweeps: one warp per atom pair, `grid` persistent CTAs of `block` threads
cudaError_t launch_nlist_96(int grid, int block, const NlistArgs &a, bool force, bool energy, bool mixed, cudaStream_t st);
cudaError_t launch_nlist_generic(int grid, int block, const NlistArgs &a, bool force, bool energy, bool mixed, cudaStream_t st);

}  // namespace scmd
