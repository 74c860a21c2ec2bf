// sc_analysis.cuh -- on-device analysis that reuses the resident state: the radial-distribution counts of the
// central atoms ("the atoms located within 3 A of the cluster center of mass were selected.
// For these atoms the RDF was calculated with a distance bin of 0.4 A"; Eq. (11) g(r) = rho(r) / rho_bar).
// The device produces the integer part -- counts[b] = ordered pairs (i reference, j != i) with
// floor(r_ij / bin_width) = b -- bit-exactly: d in binary64, r2 = fma(dz, dz, fma(dy, dy, dx*dx)), r = sqrt(r2)
// (correctly rounded), b = floor(r * (1 / bin_width)); the normalisation to g(r) is the caller's arithmetic.
#pragma once
#include "sc_device.cuh"

namespace scmd {

constexpr int kRdfMaxBins = 4096;
constexpr int kRdfBlock = 256;

#ifdef SCMD_MAIN_TU
// one block: centre of mass (equal masses) in a fixed order -> meta[0..2]
__global__ void rdf_centre_kernel(const double4 *__restrict__ xs, int N, double *__restrict__ meta) {
    __shared__ double scratch[32];
    double sx = 0.0, sy = 0.0, sz = 0.0;
    for (int i = threadIdx.x; i < N; i += blockDim.x) {
        const double4 p = xs[i];
        sx += p.x; sy += p.y; sz += p.z;
    }
    const double tx = block_sum(sx, scratch), ty = block_sum(sy, scratch), tz = block_sum(sz, scratch);
    if (threadIdx.x == 0) { meta[0] = tx / double(N); meta[1] = ty / double(N); meta[2] = tz / double(N); }
}

// reference atoms: |r_i - centre|^2 < r_select^2 (strict); their order in refs[] is arbitrary (integer result)
__global__ void rdf_select_kernel(const double4 *__restrict__ xs, int N, const double *__restrict__ meta, double rs2,
                                  int *__restrict__ refs, unsigned int *__restrict__ n_ref) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const double4 p = xs[i];
    const double ex = p.x - meta[0], ey = p.y - meta[1], ez = p.z - meta[2];
    if (fma(ez, ez, fma(ey, ey, ex * ex)) < rs2) refs[atomicAdd(n_ref, 1u)] = i;
}

// a CTA holds kRdfBlock atoms j (one per thread) and walks all reference atoms; histogram in shared memory,
// flushed with 64-bit integer atomics
__global__ void __launch_bounds__(kRdfBlock) rdf_count_kernel(const double4 *__restrict__ xs, int N,
                                                              const int *__restrict__ refs,
                                                              const unsigned int *__restrict__ n_ref_p, double inv_bin,
                                                              int n_bins, unsigned long long *__restrict__ counts) {
    __shared__ unsigned int hist[kRdfMaxBins];
    for (int b = threadIdx.x; b < n_bins; b += kRdfBlock) hist[b] = 0u;
    __syncthreads();
    const int j = blockIdx.x * kRdfBlock + threadIdx.x;
    const int n_ref = int(*n_ref_p);
    if (j < N) {
        const double4 pj = xs[j];
        for (int k = 0; k < n_ref; ++k) {
            const int i = refs[k];
            if (i == j) continue;
            const double4 pi = xs[i];
            const double dx = pi.x - pj.x, dy = pi.y - pj.y, dz = pi.z - pj.z;
            const double r = sqrt(fma(dz, dz, fma(dy, dy, dx * dx)));
            const double fb = floor(r * inv_bin);
            if (fb < double(n_bins)) atomicAdd(&hist[int(fb)], 1u);
        }
    }
    __syncthreads();
    for (int b = threadIdx.x; b < n_bins; b += kRdfBlock)
        if (hist[b]) atomicAdd(&counts[b], (unsigned long long)hist[b]);
}
#endif  // SCMD_MAIN_TU

}  // namespace scmd
