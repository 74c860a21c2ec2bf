// sc_cutoff.cuh -- the cutoff variant (BASELINE.json; the paper itself runs all pairs and names
// cutoffs as work in progress): cell binning by counting sort, Verlet neighbour
// rows with a skin, and the two list-driven sweeps.
//
// Design constraint (measured, profiles/ncu_cutoff_r1.md): a list-driven FP64 sweep on sm_100a is
// bound by L1 wavefronts (one per distinct 128-byte line a warp-wide gather touches), not by the
// FP64 pipe, unless the 32 lanes of a warp gather ADJACENT records.  Hence:
//   * atoms are sorted into FINE cells (edge = list radius / G, G = 4 by default), x fastest, so the
//     in-range neighbours of an atom are ~60 contiguous runs of the internal order;
//   * one WARP walks one neighbour row (rows are row-major, ascending in j, padded to a multiple of
//     32 with the index of a dummy record at infinity): index loads are 128 contiguous bytes and a
//     record gather touches ~1 line per 3 entries;
//   * records are fetched with one 256-bit load (SASS LDG.E.ENL2.256).
//
// rebuild_kernel: ONE cooperative launch per force evaluation.  It reads the device-side skin
// criterion (largest squared displacement since the last build, written by kick_drift_kernel) and
// returns at once when the rows are still valid, so the step loop never synchronises with the
// host.  When it does rebuild, the phases are separated by grid-wide barriers:
//   P0  zero the cell histogram; per-CTA partial sums / minima / maxima of the positions
//   P1  CTA 0: fixed-order reduction -> cell grid: edge = r_list / G with the largest G <= G_max whose
//       grid fits the cell budget, centred on the centroid, at most max_dim cells per axis; atoms
//       outside are clamped into the boundary cells (clamping is 1-Lipschitz per axis, so "within
//       r_list => at most G cells apart" stays true and evaporated atoms cost nothing)
//   P2  cell index per atom, histogram by integer atomics (slot order is arbitrary ...)
//   P3  exclusive scan of the histogram (per-CTA chunk sums, then chunk scans)
//   P4  scatter atom indices into their cell segment
//   P5  rank of every atom inside its cell by atom index (... and made canonical here: every later
//       floating-point sum runs in an order that does not depend on atomics)
//   P6  permute records, velocities, perm into cell order (into the alternate buffers)
//   P7  copy back; the records at the build become the reference for the skin criterion
//   P8  neighbour rows, one warp per atom: for each of the <= (2G+1)^2 rows of cells in y, z the
//       x-run of cells that can hold a neighbour is one contiguous range of the internal order; the
//       warp tests 32 candidates at a time and appends, in order, every j != k with
//       r^2 < (r_c + skin)^2; rows never truncate silently (overflow flag -> SC_ERR_CAPACITY)
// After a build the library's internal atom order IS the cell order; perm[k] = caller's index.
//
// nlist_kernel: LPA lanes (32 by default) walk one row, gather the 32-byte record of j, apply the
// strict binary64 test r^2 < r_c^2 (reading Q7: same decision value as the oracle) and accumulate
// the same pair terms as the all-pairs sweeps.  MIXED: pair arithmetic in binary32 on the converted
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

constexpr int kFineMax = 4;      // G_max: fine cells per list radius (the grid falls back to coarser cells
                                 // when the fine grid would exceed the cell budget)
constexpr double kFarAway = 1.0e150;   // coordinates of the dummy record that pads every neighbour row

struct CellGrid {          // written by CTA 0 in P1, read by everyone afterwards
    double ox, oy, oz;     // origin
    double inv_edge;       // 1 / cell edge
    int nx, ny, nz, ncell;
    int fine;              // G: a neighbour within the list radius is at most G cells away per axis
    int pad_;
};

struct RebuildArgs {
    double4 *xs, *xs_alt, *xs_ref;
    double *vel, *vel_alt;          // vel may be unset (have_vel == 0): then not permuted
    int *perm, *perm_alt;
    int *cell_of, *slot_of, *cell_sorted;
    int *cell_count, *cell_start;   // [ncell_max + 1]
    int *order_tmp, *order;
    int *nlist, *ncount;            // rows: nlist[k * kmax + e], ascending j, padded with n_atoms to a multiple of 32
    double *blockpart;              // [9 * gridDim.x]
    int *scanpart;                  // [gridDim.x + 1]
    CellGrid *grid;
    double *scal;
    unsigned long long *counters;
    int n_atoms, kmax, max_dim, have_vel, fine_max;
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
    // ---- decision: uniform over the grid (plain loads of values nobody writes before the last phase) ----
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
            CellGrid g;
            double com[3], half[3];
            for (int d = 0; d < 3; ++d) {
                com[d] = sh[d][0] / double(N);
                half[d] = fmax(com[d] - sh[3 + d][0], sh[6 + d][0] - com[d]);
            }
            // the finest grid (G cells per list radius) whose covering box fits the cell budget
            int G = a.fine_max;
            double edge = 0.0;
            int nc[3];
            for (;; --G) {
                edge = a.r_list / double(G) * (1.0 + 1e-6);
                double cells = 1.0;
                for (int d = 0; d < 3; ++d) {
                    double want = ceil(2.0 * half[d] / edge);
                    if (!(want >= 1.0)) want = 1.0;                  // also catches NaN
                    nc[d] = want > double(a.max_dim) ? a.max_dim : int(want);
                    cells *= want;
                }
                if (G == 1 || cells <= double(ncell_cap)) break;
            }
            g.inv_edge = 1.0 / edge;
            double org[3];
            for (int d = 0; d < 3; ++d) {
                org[d] = com[d] - 0.5 * double(nc[d]) * edge;
                if (!isfinite(org[d])) org[d] = 0.0;
            }
            g.ox = org[0]; g.oy = org[1]; g.oz = org[2];
            g.nx = nc[0]; g.ny = nc[1]; g.nz = nc[2]; g.ncell = nc[0] * nc[1] * nc[2];
            g.fine = G; g.pad_ = 0;
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

    // ---- P3: exclusive scan cell_count[0..ncell) -> cell_start[0..ncell]: CTA b owns one chunk ----
    const int nc_all = g.ncell;
    const int chunk = (nc_all + int(gridDim.x) - 1) / int(gridDim.x);
    const int cb = min(nc_all, int(blockIdx.x) * chunk), ce = min(nc_all, cb + chunk);
    {
        int s = 0;
        for (int c = cb + tid; c < ce; c += 256) s += a.cell_count[c];
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
        if (lane == 0) sh_scan[warp] = s;
        __syncthreads();
        if (tid == 0) {
            int t = 0;
            for (int w = 0; w < 8; ++w) t += sh_scan[w];
            a.scanpart[blockIdx.x] = t;
        }
    }
    grid.sync();
    {
        // offset of this CTA's chunk = sum of the chunk totals before it
        int s = 0;
        for (int b = tid; b < int(blockIdx.x); b += 256) s += a.scanpart[b];
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
        __syncthreads();
        if (lane == 0) sh_scan[warp] = s;
        __syncthreads();
        int base = 0;
        for (int w = 0; w < 8; ++w) base += sh_scan[w];
        __syncthreads();
        // chunk scan: each thread takes a contiguous piece
        const int len = ce - cb, piece = (len + 255) / 256;
        const int pb = cb + min(len, tid * piece), pe = cb + min(len, tid * piece + piece);
        int mine = 0;
        for (int c = pb; c < pe; ++c) mine += a.cell_count[c];
        sh_scan[tid] = mine;
        __syncthreads();
        if (tid == 0) {
            int run = base;
            for (int t = 0; t < 256; ++t) { const int v = sh_scan[t]; sh_scan[t] = run; run += v; }
        }
        __syncthreads();
        int run = sh_scan[tid];
        for (int c = pb; c < pe; ++c) { a.cell_start[c] = run; run += a.cell_count[c]; }
        if (gtid == 0) a.cell_start[nc_all] = N;
    }
    grid.sync();

    // ---- P4: scatter ----
    for (int i = gtid; i < N; i += gsize) a.order_tmp[a.cell_start[a.cell_of[i]] + a.slot_of[i]] = i;
    grid.sync();

    // ---- P5: rank inside the cell by atom index (one thread per slot; cells hold a few atoms) ----
    for (int k = gtid; k < N; k += gsize) {
        const int v = a.order_tmp[k];
        const int c = a.cell_of[v];
        const int b = a.cell_start[c], e = a.cell_start[c + 1];
        int rank = 0;
        for (int t = b; t < e; ++t) rank += (a.order_tmp[t] < v) ? 1 : 0;
        a.order[b + rank] = v;
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
    if (gtid == 0) a.xs[N] = make_double4(kFarAway, kFarAway, kFarAway, 0.0);   // the dummy record
    grid.sync();

    // ---- P8: neighbour rows, one warp per atom ----
    const double rl2 = a.r_list * a.r_list;
    const double rl2_cells = rl2 * g.inv_edge * g.inv_edge;           // (list radius / edge)^2
    const int G = g.fine;
    const unsigned lt_mask = (1u << lane) - 1u;
    int my_max = 0;
    const int gwarp = gtid >> 5, nwarps = gsize >> 5;
    for (int k = gwarp; k < N; k += nwarps) {
        const double4 p = a.xs[k];
        const int c = a.cell_sorted[k];
        const int cx = c % g.nx, cy = (c / g.nx) % g.ny, cz = c / (g.nx * g.ny);
        int *row = a.nlist + size_t(k) * a.kmax;
        int cnt = 0;
        for (int zz = max(cz - G, 0); zz <= min(cz + G, g.nz - 1); ++zz) {
            const int adz = max(abs(zz - cz) - 1, 0);
            for (int yy = max(cy - G, 0); yy <= min(cy + G, g.ny - 1); ++yy) {
                const int ady = max(abs(yy - cy) - 1, 0);
                // cells of this row whose nearest point can be inside the list sphere
                const double rem = rl2_cells - double(adz * adz + ady * ady);
                if (!(rem > 0.0)) continue;
                const int mx = min(G, int(sqrt(rem)) + 1);
                const int rowc = (zz * g.ny + yy) * g.nx;
                const int jb = a.cell_start[rowc + max(cx - mx, 0)], je = a.cell_start[rowc + min(cx + mx, g.nx - 1) + 1];
                for (int j0 = jb; j0 < je; j0 += 32) {
                    const int j = j0 + lane;
                    bool ok = false;
                    if (j < je) {
                        const double4 q = a.xs[j];
                        const double dx = p.x - q.x, dy = p.y - q.y, dz = p.z - q.z;
                        const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
                        ok = (r2 < rl2) && (j != k);
                    }
                    const unsigned m = __ballot_sync(0xffffffffu, ok);
                    const int at = cnt + __popc(m & lt_mask);
                    if (ok && at < a.kmax) row[at] = j;
                    cnt += __popc(m);
                }
            }
        }
        const int kept = min(cnt, a.kmax);
        const int padded = min((kept + 31) & ~31, a.kmax);
        if (kept + lane < padded) row[kept + lane] = N;                 // pad with the dummy record
        if (lane == 0) a.ncount[k] = kept;
        my_max = max(my_max, cnt);
    }
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
    double4 *xs;              // [N + 1] (x, y, z, s'), internal order; xs[N] = the dummy record at infinity
    const int *nlist;         // [N][kmax] rows, padded with N to a multiple of 32
    const int *ncount;        // [N]
    int n_atoms, kmax;
    int atoms_per_cta;        // consecutive atoms one CTA works through (multiple of 4 * 32 / LPA)
    double *rho;              // [N]    sweep 1
    double *force;            // [N*3]  sweep 2
    double *partial;          // [gridDim.x]
    unsigned long long *pairs_in_cut;   // sweep 1: += ordered pairs with r^2 < r_c^2 (zeroed by the host)
    double rc2;
    PairConsts c;
};

constexpr int kNlistBlock = 128;
constexpr int kNlistWarps = kNlistBlock / 32;
constexpr int kMixedChunk = 8;      // binary32 partial sums are flushed into binary64 every 8 row entries

// one 32-byte record with a single 256-bit load (SASS LDG.E.ENL2.256): one L1 wavefront per line touched
__device__ __forceinline__ double4 load_record(const double4 *p) {
    double4 r;
    asm volatile("ld.global.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(r.x), "=d"(r.y), "=d"(r.z), "=d"(r.w) : "l"(p));
    return r;
}

// LPA lanes per atom (32 / LPA atoms per warp at a time).  A CTA works through atoms_per_cta consecutive
// atoms of the internal (cell) order, its warps interleaved, so that the records its gathers touch stay
// in L1.
template <int LPA, int NE, int ME, bool FORCE, bool ENERGY, bool MIXED>
__global__ void __launch_bounds__(kNlistBlock) nlist_kernel(const NlistArgs a) {
    constexpr int AW = 32 / LPA;                         // atoms per warp
    __shared__ double scratch[32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int g = lane / LPA, q = lane % LPA;            // group g of the warp takes one atom, q strides its row
    const int N = a.n_atoms;
    const int n_exp = (NE > 0) ? NE : a.c.n, m_exp = (ME > 0) ? ME : a.c.m;
    const double An = a.c.An, rc2 = a.rc2;
    const float Anf = float(An);
    double contrib = 0.0;
    int npairs = 0;

    const int base = blockIdx.x * a.atoms_per_cta;
    const int end = min(N, base + a.atoms_per_cta);
    for (int i0 = base + warp * AW; i0 < end; i0 += kNlistWarps * AW) {
        const int i = i0 + g;
        const bool live = i < end;
        const int ii = live ? i : N;                     // idle groups sit on the dummy record, empty row
        const double4 pi = a.xs[ii];
        const int cnt = live ? a.ncount[i] : 0;
        const int niter = (cnt + LPA - 1) / LPA;         // rows are padded to a multiple of 32 >= LPA
        const int *row = a.nlist + size_t(live ? i : 0) * a.kmax + q;
        const float sif = float(pi.w);
        double acc0 = 0.0, acc1 = 0.0, acc2 = 0.0, acc3 = 0.0;

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
            int t = 0;
            for (; t + 3 < niter; t += 4) {                // 4 independent gathers in flight
                const int j0 = row[t * LPA], j1 = row[(t + 1) * LPA], j2 = row[(t + 2) * LPA], j3 = row[(t + 3) * LPA];
                const double4 p0 = load_record(a.xs + j0), p1 = load_record(a.xs + j1);
                const double4 p2 = load_record(a.xs + j2), p3 = load_record(a.xs + j3);
                pair(p0); pair(p1); pair(p2); pair(p3);
            }
            for (; t < niter; ++t) pair(load_record(a.xs + row[t * LPA]));
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
            int t = 0;
            for (; t + kMixedChunk - 1 < niter; t += kMixedChunk) {
                int j[kMixedChunk];
#pragma unroll
                for (int u = 0; u < kMixedChunk; ++u) j[u] = row[(t + u) * LPA];
#pragma unroll
                for (int u = 0; u < kMixedChunk; u += 4) {
                    const double4 p0 = load_record(a.xs + j[u]), p1 = load_record(a.xs + j[u + 1]);
                    const double4 p2 = load_record(a.xs + j[u + 2]), p3 = load_record(a.xs + j[u + 3]);
                    pair(p0); pair(p1); pair(p2); pair(p3);
                }
                flush();
            }
            for (; t < niter; ++t) pair(load_record(a.xs + row[t * LPA]));
            flush();
        }

        // ---- reduce over the LPA lanes of the atom (fixed order) ----
        acc0 = group_sum<LPA>(acc0);
        if constexpr (FORCE) {
            acc1 = group_sum<LPA>(acc1);
            acc2 = group_sum<LPA>(acc2);
            if constexpr (ENERGY) acc3 = group_sum<LPA>(acc3);
        }
        if (live && q == 0) {
            if constexpr (!FORCE) {
                const double rho = a.c.am * acc0;
                a.rho[i] = rho;
                const double root = rho > 0.0 ? sqrt(rho) : 0.0;           // reading Q9
                a.xs[i].w = rho > 0.0 ? a.c.Bm / root : 0.0;
                contrib += root;
            } else {
                a.force[3 * size_t(i)] = acc0;
                a.force[3 * size_t(i) + 1] = acc1;
                a.force[3 * size_t(i) + 2] = acc2;
                contrib += acc3;
            }
        }
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
