// sc_cutoff.cuh -- the cutoff variant (BASELINE.json; the paper itself runs all pairs and names
// cutoffs as work in progress): cell binning by counting sort, Verlet neighbour
// rows with a skin, and the two list-driven sweeps.
//
// rebuild_kernel: ONE cooperative launch per force evaluation.  It reads the device-side skin
// criterion (largest squared displacement since the last build, written by kick_drift_kernel) and
// returns at once when the rows are still valid, so the step loop never synchronises with the
// host.  When it does rebuild, the phases are separated by grid-wide barriers:
//   P0  zero the cell histogram; per-CTA partial sums / minima / maxima of the positions
//   P1  CTA 0: fixed-order reduction -> cell grid (edge >= r_c + skin, centred on the centroid,
//       at most max_dim cells per axis; atoms outside are clamped into the boundary cells, which
//       keeps "within r_list => adjacent cells" true, so evaporated atoms cost nothing)
//   P2  cell index per atom, histogram by integer atomics (slot order is arbitrary ...)
//   P3  CTA 0: exclusive scan of the histogram
//   P4  scatter atom indices into their cell segment
//   P5  one warp per cell: rank sort of the segment by atom index (... and made canonical here:
//       every later floating-point sum runs in an order that does not depend on atomics)
//   P6  permute records, velocities, perm into cell order (into the alternate buffers)
//   P7  copy back; the records at the build become the reference for the skin criterion
//   P8  neighbour rows: atom k scans the <= 27 neighbouring cells (3 x-adjacent cells are one
//       contiguous run in cell order) and appends every j != k with r^2 < (r_c + skin)^2 to
//       nlist[count * npad + k]; rows never truncate silently (overflow flag -> SC_ERR_CAPACITY)
// After a build the library's internal atom order IS the cell order; perm[k] = caller's index.
//
// nlist_kernel: TPA lanes per atom walk the row, gather the 32-byte record of j, apply the strict
// binary64 test r^2 < r_c^2 (reading Q7: same decision value as the oracle) and accumulate the
// same pair terms as the all-pairs sweeps.  MIXED: pair arithmetic in binary32 on the converted
// binary64 difference, accumulated in binary32 over a short chunk and flushed into binary64.
#pragma once
#include <cooperative_groups.h>

#include "sc_allpairs.cuh"
#include "sc_device.cuh"
#include "sc_integrate.cuh"

namespace scmd {
namespace cg = cooperative_groups;

enum CounterSlot {
    kCntRebuilds = 0,     // list builds since sc_create
    kCntMaxRow = 1,       // longest neighbour row at the last build
    kCntOverflow = 2,     // != 0: a row exceeded kmax at some build
    kCntListValid = 3,    // 0 forces a build at the next evaluation
    kCntPairsInCut = 4,   // ordered pairs with r^2 < r_c^2 at the last density sweep
    kNumCounters = 8
};

struct CellGrid {          // written by CTA 0 in P1, read by everyone afterwards
    double ox, oy, oz;     // origin
    double inv_edge;       // 1 / cell edge
    int nx, ny, nz, ncell;
};

struct RebuildArgs {
    double4 *xs, *xs_alt, *xs_ref;
    double *vel, *vel_alt;          // vel may be unset (have_vel == 0): then not permuted
    int *perm, *perm_alt;
    int *cell_of, *slot_of, *cell_sorted;
    int *cell_count, *cell_start;   // [ncell_max + 1]
    int *order_tmp, *order;
    int *nlist, *ncount;
    double *blockpart;              // [9 * gridDim.x]
    CellGrid *grid;
    double *scal;
    unsigned long long *counters;
    int n_atoms, npad, kmax, max_dim, have_vel;
    double r_list, half_skin2;
};

#ifdef SCMD_MAIN_TU
__device__ __forceinline__ int cell_coord(double x, double o, double inv_edge, int n) {
    const double t = (x - o) * inv_edge;
    int c = t <= 0.0 ? 0 : (t >= double(n) ? n - 1 : int(t));
    return c > n - 1 ? n - 1 : c;
}

__global__ void __launch_bounds__(256) rebuild_kernel(const RebuildArgs a) {
    cg::grid_group grid = cg::this_grid();
    const int N = a.n_atoms;
    // ---- decision: uniform over the grid (plain loads of values nobody writes before P8) ----
    const bool need = (a.counters[kCntListValid] == 0ull) || (a.scal[kSlotMaxDisp2] > a.half_skin2);
    if (!need) return;

    __shared__ double sh[9][8];
    __shared__ int sh_scan[256];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int gtid = blockIdx.x * blockDim.x + tid, gsize = gridDim.x * blockDim.x;
    const int ncell_cap = a.max_dim * a.max_dim * a.max_dim;

    // ---- P0 ----
    for (int c = gtid; c <= ncell_cap; c += gsize) a.cell_count[c] = 0;
    {
        double sx = 0, sy = 0, sz = 0, lx = 1e300, ly = 1e300, lz = 1e300, hx = -1e300, hy = -1e300, hz = -1e300;
        for (int i = gtid; i < N; i += gsize) {
            const double4 p = a.xs[i];
            sx += p.x; sy += p.y; sz += p.z;
            lx = fmin(lx, p.x); ly = fmin(ly, p.y); lz = fmin(lz, p.z);
            hx = fmax(hx, p.x); hy = fmax(hy, p.y); hz = fmax(hz, p.z);
        }
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) {
            sx += __shfl_xor_sync(0xffffffffu, sx, off); sy += __shfl_xor_sync(0xffffffffu, sy, off);
            sz += __shfl_xor_sync(0xffffffffu, sz, off);
            lx = fmin(lx, __shfl_xor_sync(0xffffffffu, lx, off)); ly = fmin(ly, __shfl_xor_sync(0xffffffffu, ly, off));
            lz = fmin(lz, __shfl_xor_sync(0xffffffffu, lz, off));
            hx = fmax(hx, __shfl_xor_sync(0xffffffffu, hx, off)); hy = fmax(hy, __shfl_xor_sync(0xffffffffu, hy, off));
            hz = fmax(hz, __shfl_xor_sync(0xffffffffu, hz, off));
        }
        if (lane == 0) {
            sh[0][warp] = sx; sh[1][warp] = sy; sh[2][warp] = sz; sh[3][warp] = lx; sh[4][warp] = ly;
            sh[5][warp] = lz; sh[6][warp] = hx; sh[7][warp] = hy; sh[8][warp] = hz;
        }
        __syncthreads();
        if (tid < 9) {
            double v = sh[tid][0];
            for (int w = 1; w < 8; ++w) v = tid < 3 ? v + sh[tid][w] : (tid < 6 ? fmin(v, sh[tid][w]) : fmax(v, sh[tid][w]));
            a.blockpart[9 * blockIdx.x + tid] = v;
        }
    }
    grid.sync();

    // ---- P1: CTA 0 builds the cell grid ----
    if (blockIdx.x == 0) {
        if (tid < 9) {
            double v = a.blockpart[tid];
            for (int b = 1; b < int(gridDim.x); ++b) {
                const double o = a.blockpart[9 * b + tid];
                v = tid < 3 ? v + o : (tid < 6 ? fmin(v, o) : fmax(v, o));
            }
            sh[tid][0] = v;
        }
        __syncthreads();
        if (tid == 0) {
            const double edge = a.r_list * (1.0 + 1e-6);
            CellGrid g;
            g.inv_edge = 1.0 / edge;
            double com[3], lo[3], hi[3], org[3];
            int nc[3];
            for (int d = 0; d < 3; ++d) {
                com[d] = sh[d][0] / double(N); lo[d] = sh[3 + d][0]; hi[d] = sh[6 + d][0];
                // cells needed to cover [lo, hi] symmetrically about the centroid, capped
                const double half = fmax(com[d] - lo[d], hi[d] - com[d]);
                double want = ceil(2.0 * half / edge);
                if (!(want >= 1.0)) want = 1.0;                      // also catches NaN
                nc[d] = want > double(a.max_dim) ? a.max_dim : int(want);
                org[d] = com[d] - 0.5 * double(nc[d]) * edge;
                if (!isfinite(org[d])) org[d] = 0.0;
            }
            g.ox = org[0]; g.oy = org[1]; g.oz = org[2];
            g.nx = nc[0]; g.ny = nc[1]; g.nz = nc[2]; g.ncell = nc[0] * nc[1] * nc[2];
            *a.grid = g;
        }
    }
    grid.sync();
    const CellGrid g = *a.grid;

    // ---- P2: cell index + histogram ----
    for (int i = gtid; i < N; i += gsize) {
        const double4 p = a.xs[i];
        const int cx = cell_coord(p.x, g.ox, g.inv_edge, g.nx);
        const int cy = cell_coord(p.y, g.oy, g.inv_edge, g.ny);
        const int cz = cell_coord(p.z, g.oz, g.inv_edge, g.nz);
        const int c = (cz * g.ny + cy) * g.nx + cx;
        a.cell_of[i] = c;
        a.slot_of[i] = atomicAdd(&a.cell_count[c], 1);
    }
    grid.sync();

    // ---- P3: CTA 0: exclusive scan cell_count[0..ncell) -> cell_start[0..ncell] ----
    if (blockIdx.x == 0) {
        const int nc = g.ncell;
        const int chunk = (nc + 255) / 256;
        const int b = tid * chunk, e = min(nc, b + chunk);
        int s = 0;
        for (int c = b; c < e; ++c) s += a.cell_count[c];
        sh_scan[tid] = s;
        __syncthreads();
        if (tid == 0) {
            int run = 0;
            for (int t = 0; t < 256; ++t) { const int v = sh_scan[t]; sh_scan[t] = run; run += v; }
        }
        __syncthreads();
        int run = sh_scan[tid];
        for (int c = b; c < e; ++c) { a.cell_start[c] = run; run += a.cell_count[c]; }
        if (tid == 0) a.cell_start[nc] = N;
    }
    grid.sync();

    // ---- P4: scatter ----
    for (int i = gtid; i < N; i += gsize) a.order_tmp[a.cell_start[a.cell_of[i]] + a.slot_of[i]] = i;
    grid.sync();

    // ---- P5: rank sort inside each cell (one warp per cell) ----
    {
        const int gwarp = gtid >> 5, nwarps = gsize >> 5;
        for (int c = gwarp; c < g.ncell; c += nwarps) {
            const int b = a.cell_start[c], e = a.cell_start[c + 1];
            for (int k = b + lane; k < e; k += 32) {
                const int v = a.order_tmp[k];
                int rank = 0;
                for (int t = b; t < e; ++t) rank += (a.order_tmp[t] < v) ? 1 : 0;
                a.order[b + rank] = v;
            }
        }
    }
    grid.sync();

    // ---- P6: permute into the alternate buffers ----
    for (int k = gtid; k < N; k += gsize) {
        const int src = a.order[k];
        a.xs_alt[k] = a.xs[src];
        a.perm_alt[k] = a.perm[src];
        a.cell_sorted[k] = a.cell_of[src];
        if (a.have_vel) {
            a.vel_alt[3 * size_t(k)] = a.vel[3 * size_t(src)];
            a.vel_alt[3 * size_t(k) + 1] = a.vel[3 * size_t(src) + 1];
            a.vel_alt[3 * size_t(k) + 2] = a.vel[3 * size_t(src) + 2];
        }
    }
    grid.sync();

    // ---- P7: copy back ----
    for (int k = gtid; k < N; k += gsize) {
        const double4 p = a.xs_alt[k];
        a.xs[k] = p;
        a.xs_ref[k] = p;
        a.perm[k] = a.perm_alt[k];
        if (a.have_vel) {
            a.vel[3 * size_t(k)] = a.vel_alt[3 * size_t(k)];
            a.vel[3 * size_t(k) + 1] = a.vel_alt[3 * size_t(k) + 1];
            a.vel[3 * size_t(k) + 2] = a.vel_alt[3 * size_t(k) + 2];
        }
    }
    grid.sync();

    // ---- P8: neighbour rows ----
    const double rl2 = a.r_list * a.r_list;
    int my_max = 0;
    for (int k = gtid; k < N; k += gsize) {
        const double4 p = a.xs[k];
        const int c = a.cell_sorted[k];
        const int cx = c % g.nx, cy = (c / g.nx) % g.ny, cz = c / (g.nx * g.ny);
        const int x0 = max(cx - 1, 0), x1 = min(cx + 1, g.nx - 1);
        int cnt = 0;
        for (int zz = max(cz - 1, 0); zz <= min(cz + 1, g.nz - 1); ++zz)
            for (int yy = max(cy - 1, 0); yy <= min(cy + 1, g.ny - 1); ++yy) {
                const int rowc = (zz * g.ny + yy) * g.nx;
                const int jb = a.cell_start[rowc + x0], je = a.cell_start[rowc + x1 + 1];
                for (int j = jb; j < je; ++j) {
                    const double4 q = a.xs[j];
                    const double dx = p.x - q.x, dy = p.y - q.y, dz = p.z - q.z;
                    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
                    if (r2 < rl2 && j != k) {
                        if (cnt < a.kmax) a.nlist[size_t(cnt) * a.npad + k] = j;
                        ++cnt;
                    }
                }
            }
        a.ncount[k] = min(cnt, a.kmax);
        my_max = max(my_max, cnt);
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) my_max = max(my_max, __shfl_xor_sync(0xffffffffu, my_max, off));
    if (lane == 0 && my_max > a.kmax) atomicExch(&a.counters[kCntOverflow], 1ull);
    // counters[kCntMaxRow] is reset below by the one thread that also bumps the build count; a max
    // across the grid needs the reset to happen first, so it lives in its own slot pair:
    if (lane == 0) atomicMax(&a.counters[kNumCounters - 1], (unsigned long long)my_max);
    grid.sync();
    if (gtid == 0) {
        a.counters[kCntMaxRow] = a.counters[kNumCounters - 1];
        a.counters[kNumCounters - 1] = 0ull;
        a.counters[kCntRebuilds] += 1ull;
        a.counters[kCntListValid] = 1ull;
        a.scal[kSlotMaxDisp2] = 0.0;
    }
}

#endif  // SCMD_MAIN_TU

// --------------------------------------------------------------------------------------------
// list-driven sweeps
// --------------------------------------------------------------------------------------------
struct NlistArgs {
    double4 *xs;              // [N] (x, y, z, s'), internal order
    const int *nlist;         // [kmax][npad]
    const int *ncount;        // [N]
    int n_atoms, npad;
    double *rho;              // [N]    sweep 1
    double *force;            // [N*3]  sweep 2
    double *partial;          // [gridDim.x]
    unsigned long long *pairs_in_cut;   // sweep 1: += ordered pairs with r^2 < r_c^2 (zeroed by the host)
    double rc2;
    PairConsts c;
};

constexpr int kNlistBlock = 128;
constexpr int kMixedChunk = 8;      // binary32 partial sums are flushed into binary64 every 8 row entries

template <int TPA, int NE, int ME, bool FORCE, bool ENERGY, bool MIXED>
__global__ void __launch_bounds__(kNlistBlock) nlist_kernel(const NlistArgs a) {
    constexpr int AW = 32 / TPA;                         // atoms per warp
    __shared__ double scratch[32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int al = lane % AW, q = lane / AW;
    const int N = a.n_atoms;
    const int i = (blockIdx.x * (kNlistBlock / 32) + warp) * AW + al;
    const bool live = i < N;
    const int ii = live ? i : N - 1;
    const double4 pi = a.xs[ii];
    const int cnt = live ? a.ncount[ii] : 0;
    const int n_exp = (NE > 0) ? NE : a.c.n, m_exp = (ME > 0) ? ME : a.c.m;
    const double An = a.c.An, rc2 = a.rc2;
    const float Anf = float(An);
    const float sif = float(pi.w);
    double acc0 = 0.0, acc1 = 0.0, acc2 = 0.0, acc3 = 0.0;
    int npairs = 0;
    const int *row = a.nlist + ii;

    if constexpr (!MIXED) {
        auto pair = [&](const double4 &p) {
            const double dx = pi.x - p.x, dy = pi.y - p.y, dz = pi.z - p.z;
            const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
            if (r2 < rc2) {
                if constexpr (!FORCE) {
                    ++npairs;
                    if constexpr (ME > 0 && ME % 2 == 0) {
                        const double w = rcp_fast(r2);
                        if constexpr (ME == 6) acc0 = fma(w * w, w, acc0);
                        else acc0 += ipow_c<ME / 2>(w);
                    } else if constexpr (ME > 0) {
                        acc0 += ipow_c<ME>(rsqrt_fast(r2));
                    } else {
                        acc0 += ipow_rt(rsqrt_fast(r2), m_exp);
                    }
                } else {
                    const double y = rsqrt_fast(r2);
                    const double w = y * y;
                    const double ss = pi.w + p.w;
                    double coef;
                    if constexpr (NE == 9 && ME == 6) {
                        const double w2 = w * w, w4 = w2 * w2, y3 = w * y;
                        coef = w4 * fma(An, y3, -ss);
                        if constexpr (ENERGY) acc3 = fma(w4, y, acc3);
                    } else {
                        const double pm = (ME > 0) ? ipow_c<ME>(y) : ipow_rt(y, m_exp);
                        const double pn = (NE > 0) ? ipow_c<NE>(y) : ipow_rt(y, n_exp);
                        coef = w * fma(An, pn, -ss * pm);
                        if constexpr (ENERGY) acc3 += pn;
                    }
                    acc0 = fma(coef, dx, acc0);
                    acc1 = fma(coef, dy, acc1);
                    acc2 = fma(coef, dz, acc2);
                }
            }
        };
        int k = q;
        for (; k + 3 * TPA < cnt; k += 4 * TPA) {          // 4 independent gathers in flight
            const int j0 = row[size_t(k) * a.npad], j1 = row[size_t(k + TPA) * a.npad];
            const int j2 = row[size_t(k + 2 * TPA) * a.npad], j3 = row[size_t(k + 3 * TPA) * a.npad];
            const double4 p0 = a.xs[j0], p1 = a.xs[j1], p2 = a.xs[j2], p3 = a.xs[j3];
            pair(p0); pair(p1); pair(p2); pair(p3);
        }
        for (; k < cnt; k += TPA) pair(a.xs[row[size_t(k) * a.npad]]);
    } else {
        float f0 = 0.f, f1 = 0.f, f2 = 0.f, f3 = 0.f;
        auto pair = [&](const double4 &p) {
            const double dxd = pi.x - p.x, dyd = pi.y - p.y, dzd = pi.z - p.z;
            const double r2d = fma(dzd, dzd, fma(dyd, dyd, dxd * dxd));
            if (r2d < rc2) {                                   // membership decided in binary64 (Q7)
                const float dx = float(dxd), dy = float(dyd), dz = float(dzd);
                const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                if constexpr (!FORCE) {
                    ++npairs;
                    if constexpr (ME > 0 && ME % 2 == 0) {
                        const float w = rcp_fast_f(r2);
                        if constexpr (ME == 6) f0 = fmaf(w * w, w, f0);
                        else f0 += ipow_cf<ME / 2>(w);
                    } else if constexpr (ME > 0) {
                        f0 += ipow_cf<ME>(rsqrt_fast_f(r2));
                    } else {
                        f0 += ipow_rtf(rsqrt_fast_f(r2), m_exp);
                    }
                } else {
                    const float y = rsqrt_fast_f(r2);
                    const float w = y * y;
                    const float ss = sif + float(p.w);
                    float coef;
                    if constexpr (NE == 9 && ME == 6) {
                        const float w2 = w * w, w4 = w2 * w2, y3 = w * y;
                        coef = w4 * fmaf(Anf, y3, -ss);
                        if constexpr (ENERGY) f3 = fmaf(w4, y, f3);
                    } else {
                        const float pm = (ME > 0) ? ipow_cf<ME>(y) : ipow_rtf(y, m_exp);
                        const float pn = (NE > 0) ? ipow_cf<NE>(y) : ipow_rtf(y, n_exp);
                        coef = w * fmaf(Anf, pn, -ss * pm);
                        if constexpr (ENERGY) f3 += pn;
                    }
                    f0 = fmaf(coef, dx, f0);
                    f1 = fmaf(coef, dy, f1);
                    f2 = fmaf(coef, dz, f2);
                }
            }
        };
        auto flush = [&]() {
            acc0 += double(f0); f0 = 0.f;
            if constexpr (FORCE) {
                acc1 += double(f1); acc2 += double(f2); f1 = f2 = 0.f;
                if constexpr (ENERGY) { acc3 += double(f3); f3 = 0.f; }
            }
        };
        int k = q;
        for (; k + (kMixedChunk - 1) * TPA < cnt; k += kMixedChunk * TPA) {
            int j[kMixedChunk];
#pragma unroll
            for (int u = 0; u < kMixedChunk; ++u) j[u] = row[size_t(k + u * TPA) * a.npad];
#pragma unroll
            for (int u = 0; u < kMixedChunk; u += 4) {
                const double4 p0 = a.xs[j[u]], p1 = a.xs[j[u + 1]], p2 = a.xs[j[u + 2]], p3 = a.xs[j[u + 3]];
                pair(p0); pair(p1); pair(p2); pair(p3);
            }
            flush();
        }
        for (; k < cnt; k += TPA) pair(a.xs[row[size_t(k) * a.npad]]);
        flush();
    }

    // ---- reduce over the TPA lanes of an atom (lanes al, al + AW, al + 2 AW, ...) ----
#pragma unroll
    for (int off = AW; off < 32; off <<= 1) {
        acc0 += __shfl_xor_sync(0xffffffffu, acc0, off);
        if constexpr (FORCE) {
            acc1 += __shfl_xor_sync(0xffffffffu, acc1, off);
            acc2 += __shfl_xor_sync(0xffffffffu, acc2, off);
            if constexpr (ENERGY) acc3 += __shfl_xor_sync(0xffffffffu, acc3, off);
        } else {
            npairs += __shfl_xor_sync(0xffffffffu, npairs, off);
        }
    }
    double contrib = 0.0;
    if (live && q == 0) {
        if constexpr (!FORCE) {
            const double rho = a.c.am * acc0;
            a.rho[i] = rho;
            const double root = rho > 0.0 ? sqrt(rho) : 0.0;           // reading Q9
            a.xs[i].w = rho > 0.0 ? a.c.Bm / root : 0.0;
            contrib = root;
        } else {
            a.force[3 * size_t(i)] = acc0;
            a.force[3 * size_t(i) + 1] = acc1;
            a.force[3 * size_t(i) + 2] = acc2;
            contrib = acc3;
        }
    } else {
        npairs = 0;
    }
    if constexpr (!FORCE) {
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) npairs += __shfl_xor_sync(0xffffffffu, npairs, off);
        if (lane == 0 && npairs) atomicAdd(a.pairs_in_cut, (unsigned long long)npairs);
    }
    if (a.partial) {
        const double t = block_sum(contrib, scratch);
        if (threadIdx.x == 0) a.partial[blockIdx.x] = t;
    }
}

#ifdef SCMD_MAIN_TU
// caller's order <-> internal order at the boundary
__global__ void scatter_by_perm_kernel(const double *__restrict__ src, double *__restrict__ dst,
                                       const int *__restrict__ perm, int N, int width) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < N) {
        const size_t o = size_t(perm[k]) * width, s = size_t(k) * width;
        for (int c = 0; c < width; ++c) dst[o + c] = src[s + c];
    }
}
__global__ void unpack_positions_perm_kernel(const double4 *__restrict__ xs, double *__restrict__ pos,
                                             const int *__restrict__ perm, int N) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < N) {
        const double4 p = xs[k];
        const size_t o = 3 * size_t(perm[k]);
        pos[o] = p.x; pos[o + 1] = p.y; pos[o + 2] = p.z;
    }
}
__global__ void iota_kernel(int *__restrict__ perm, int N) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < N) perm[k] = k;
}
__global__ void reset_list_state_kernel(unsigned long long *__restrict__ counters, double *__restrict__ scal) {
    counters[kCntListValid] = 0ull;
    scal[kSlotMaxDisp2] = 0.0;
}
__global__ void zero_u64_kernel(unsigned long long *p) { *p = 0ull; }
#endif  // SCMD_MAIN_TU

}  // namespace scmd
