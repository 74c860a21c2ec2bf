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

// ---------------------------------------------------------------------------------------------
// Mean-square displacement for Eq. (12): "cluster was translated and rotated as a whole in
// order to minimize the root-mean-square displacement of atoms from a reference structure ... the diffusion
// coefficient was calculated for all atoms located within 10 A of the cluster center of mass".
// x_i = current positions (resident records), y_i = reference structure (caller's device array, caller's atom
// order; `perm` maps the internal index to it on the list path, NULL = identity).  Five small launches, all sums
// in a fixed order (per-CTA partials, then one thread per component):
//   centroids -> 3x3 covariance of the centred sets -> rotation (one thread: Horn's 4x4 symmetric matrix, cyclic
//   Jacobi, largest eigenvalue's unit quaternion) -> sum of |R x_i' - y_i'|^2 over the selected atoms -> total.
// meta: [0..2] centroid of x used, [3..5] centroid of y, [6..14] R row-major, [15] sum, [16] count.
// ---------------------------------------------------------------------------------------------
constexpr int kMsdBlock = 256;
constexpr int kMsdMaxBlocks = 512;
constexpr int kMsdPartStride = 9;          // doubles per CTA in each of the three partial regions
constexpr int kMsdMeta = 32;

__device__ __forceinline__ void msd_load_ref(const double *__restrict__ ref, const int *__restrict__ perm, int k,
                                             double &x, double &y, double &z) {
    const size_t o = 3 * size_t(perm ? perm[k] : k);
    x = ref[o]; y = ref[o + 1]; z = ref[o + 2];
}

__global__ void __launch_bounds__(kMsdBlock) msd_centroid_kernel(const double4 *__restrict__ xs, const double *__restrict__ ref,
                                                                 const int *__restrict__ perm, int N, double *__restrict__ part) {
    __shared__ double scratch[32];
    double s[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    for (int k = blockIdx.x * kMsdBlock + threadIdx.x; k < N; k += gridDim.x * kMsdBlock) {
        const double4 p = xs[k];
        double rx, ry, rz;
        msd_load_ref(ref, perm, k, rx, ry, rz);
        s[0] += p.x; s[1] += p.y; s[2] += p.z; s[3] += rx; s[4] += ry; s[5] += rz;
    }
#pragma unroll
    for (int q = 0; q < 6; ++q) {
        const double t = block_sum(s[q], scratch);
        if (threadIdx.x == 0) part[blockIdx.x * kMsdPartStride + q] = t;
    }
}

// every CTA re-derives the centroids from the partials (same order everywhere), CTA 0 publishes them
__global__ void __launch_bounds__(kMsdBlock) msd_covariance_kernel(const double4 *__restrict__ xs, const double *__restrict__ ref,
                                                                   const int *__restrict__ perm, int N, int align,
                                                                   const double *__restrict__ part_in, double *__restrict__ part_out,
                                                                   double *__restrict__ meta) {
    __shared__ double scratch[32];
    __shared__ double cen[6];
    if (threadIdx.x < 6) {
        double t = 0.0;
        for (int b = 0; b < int(gridDim.x); ++b) t += part_in[b * kMsdPartStride + threadIdx.x];
        cen[threadIdx.x] = t / double(N);
    }
    __syncthreads();
    if (threadIdx.x < 3 && align == 0) cen[threadIdx.x] = cen[3 + threadIdx.x];      // no fit: both sets about the reference centroid
    __syncthreads();
    if (blockIdx.x == 0 && threadIdx.x < 6) meta[threadIdx.x] = cen[threadIdx.x];
    double s[9];
#pragma unroll
    for (int q = 0; q < 9; ++q) s[q] = 0.0;
    for (int k = blockIdx.x * kMsdBlock + threadIdx.x; k < N; k += gridDim.x * kMsdBlock) {
        const double4 p = xs[k];
        double rx, ry, rz;
        msd_load_ref(ref, perm, k, rx, ry, rz);
        const double x[3] = {p.x - cen[0], p.y - cen[1], p.z - cen[2]};
        const double y[3] = {rx - cen[3], ry - cen[4], rz - cen[5]};
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int b = 0; b < 3; ++b) s[3 * a + b] = fma(x[a], y[b], s[3 * a + b]);     // S_ab = sum_i x'_ia y'_ib
    }
#pragma unroll
    for (int q = 0; q < 9; ++q) {
        const double t = block_sum(s[q], scratch);
        if (threadIdx.x == 0) part_out[blockIdx.x * kMsdPartStride + q] = t;
    }
}

// one warp: threads 0..8 total the covariance, thread 0 solves for the rotation
__global__ void msd_rotation_kernel(const double *__restrict__ part, int n_blocks, int align, double *__restrict__ meta) {
    __shared__ double S[9];
    if (threadIdx.x < 9) {
        double t = 0.0;
        for (int b = 0; b < n_blocks; ++b) t += part[b * kMsdPartStride + threadIdx.x];
        S[threadIdx.x] = t;
    }
    __syncwarp();
    if (threadIdx.x != 0) return;
    double R[9] = {1.0, 0.0, 0.0, 0.0, 1.0, 0.0, 0.0, 0.0, 1.0};
    if (align >= 2) {
        const double Sxx = S[0], Sxy = S[1], Sxz = S[2], Syx = S[3], Syy = S[4], Syz = S[5], Szx = S[6], Szy = S[7], Szz = S[8];
        // Horn (1987): the unit quaternion that maximises sum_i y_i' . (R x_i') is the eigenvector of the largest
        // eigenvalue of this symmetric matrix
        double A[4][4] = {{Sxx + Syy + Szz, Syz - Szy, Szx - Sxz, Sxy - Syx},
                          {Syz - Szy, Sxx - Syy - Szz, Sxy + Syx, Szx + Sxz},
                          {Szx - Sxz, Sxy + Syx, -Sxx + Syy - Szz, Syz + Szy},
                          {Sxy - Syx, Szx + Sxz, Syz + Szy, -Sxx - Syy + Szz}};
        double V[4][4] = {{1.0, 0.0, 0.0, 0.0}, {0.0, 1.0, 0.0, 0.0}, {0.0, 0.0, 1.0, 0.0}, {0.0, 0.0, 0.0, 1.0}};
        double scale = 0.0;
        for (int p = 0; p < 4; ++p)
            for (int q = 0; q < 4; ++q) scale += A[p][q] * A[p][q];
        for (int sweep = 0; sweep < 40; ++sweep) {
            double off = 0.0;
            for (int p = 0; p < 4; ++p)
                for (int q = p + 1; q < 4; ++q) off += A[p][q] * A[p][q];
            if (!(off > 1e-40 * scale)) break;
            for (int p = 0; p < 4; ++p)
                for (int q = p + 1; q < 4; ++q) {
                    const double apq = A[p][q];
                    if (apq == 0.0) continue;
                    const double theta = (A[q][q] - A[p][p]) / (2.0 * apq);
                    const double t = (theta >= 0.0 ? 1.0 : -1.0) / (fabs(theta) + sqrt(theta * theta + 1.0));
                    const double cs = 1.0 / sqrt(t * t + 1.0), sn = t * cs;
                    for (int k = 0; k < 4; ++k) {              // columns p, q
                        const double akp = A[k][p], akq = A[k][q];
                        A[k][p] = cs * akp - sn * akq;
                        A[k][q] = sn * akp + cs * akq;
                    }
                    for (int k = 0; k < 4; ++k) {              // rows p, q
                        const double apk = A[p][k], aqk = A[q][k];
                        A[p][k] = cs * apk - sn * aqk;
                        A[q][k] = sn * apk + cs * aqk;
                    }
                    for (int k = 0; k < 4; ++k) {
                        const double vkp = V[k][p], vkq = V[k][q];
                        V[k][p] = cs * vkp - sn * vkq;
                        V[k][q] = sn * vkp + cs * vkq;
                    }
                }
        }
        int best = 0;
        for (int p = 1; p < 4; ++p)
            if (A[p][p] > A[best][best]) best = p;
        double a = V[0][best], b = V[1][best], c = V[2][best], d = V[3][best];
        const double nrm = sqrt(a * a + b * b + c * c + d * d);
        a /= nrm; b /= nrm; c /= nrm; d /= nrm;
        R[0] = a * a + b * b - c * c - d * d; R[1] = 2.0 * (b * c - a * d);           R[2] = 2.0 * (b * d + a * c);
        R[3] = 2.0 * (b * c + a * d);         R[4] = a * a - b * b + c * c - d * d;   R[5] = 2.0 * (c * d - a * b);
        R[6] = 2.0 * (b * d - a * c);         R[7] = 2.0 * (c * d + a * b);           R[8] = a * a - b * b - c * c + d * d;
    }
    for (int q = 0; q < 9; ++q) meta[6 + q] = R[q];
}

// selection: reference position strictly within r_centre of the reference centroid (rc2 <= 0: every atom)
__global__ void __launch_bounds__(kMsdBlock) msd_accumulate_kernel(const double4 *__restrict__ xs, const double *__restrict__ ref,
                                                                   const int *__restrict__ perm, int N, double rc2,
                                                                   const double *__restrict__ meta, double *__restrict__ part) {
    __shared__ double scratch[32];
    __shared__ double m[15];
    if (threadIdx.x < 15) m[threadIdx.x] = meta[threadIdx.x];
    __syncthreads();
    double sum = 0.0, cnt = 0.0;
    for (int k = blockIdx.x * kMsdBlock + threadIdx.x; k < N; k += gridDim.x * kMsdBlock) {
        const double4 p = xs[k];
        double rx, ry, rz;
        msd_load_ref(ref, perm, k, rx, ry, rz);
        const double x0 = p.x - m[0], x1 = p.y - m[1], x2 = p.z - m[2];
        const double y0 = rx - m[3], y1 = ry - m[4], y2 = rz - m[5];
        const bool sel = !(rc2 > 0.0) || (y0 * y0 + y1 * y1 + y2 * y2 < rc2);
        const double d0 = fma(m[6], x0, fma(m[7], x1, m[8] * x2)) - y0;
        const double d1 = fma(m[9], x0, fma(m[10], x1, m[11] * x2)) - y1;
        const double d2 = fma(m[12], x0, fma(m[13], x1, m[14] * x2)) - y2;
        if (sel) { sum += fma(d2, d2, fma(d1, d1, d0 * d0)); cnt += 1.0; }
    }
    const double ts = block_sum(sum, scratch), tc = block_sum(cnt, scratch);
    if (threadIdx.x == 0) { part[blockIdx.x * kMsdPartStride] = ts; part[blockIdx.x * kMsdPartStride + 1] = tc; }
}

__global__ void msd_total_kernel(const double *__restrict__ part, int n_blocks, double *__restrict__ meta) {
    if (threadIdx.x < 2) {
        double t = 0.0;
        for (int b = 0; b < n_blocks; ++b) t += part[b * kMsdPartStride + threadIdx.x];
        meta[15 + threadIdx.x] = t;
    }
}
#endif  // SCMD_MAIN_TU

}  // namespace scmd
