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
// the same pair terms as the all-pairs sweeps.  MIXED: the rows gather split binary32 records (x = xh + xl)
// and the whole pair term runs in binary32 -- no conversion, no binary64 instruction -- except that an entry
// whose binary32 r^2 lies within 2e-6 r_c^2 of the cutoff takes its set-membership decision from the binary64
// records (reading Q7: membership is the oracle's, bit for bit); partial sums are flushed into binary64 after
// every batch.
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
constexpr float kFarAwayF = 1.0e18f;   // ... of its binary32 twin (its r^2 = 3e36 stays finite)

struct CellGrid {          // written by CTA 0 in P1, read by everyone afterwards
    double ox, oy, oz;     // origin
    double inv_edge;       // 1 / cell edge
    int nx, ny, nz, ncell;
    int fine;              // G: a neighbour within the list radius is at most G cells away per axis
    int pad_;
};

struct RebuildArgs {
    double4 *xs, *xs_alt, *xs_ref;
    RecF *xfr;                      // mixed list sweeps: split binary32 records in internal order (else NULL)
    double *vel, *vel_alt;          // vel may be unset (have_vel == 0): then not permuted
    int *perm, *perm_alt;
    int *cell_of, *slot_of, *cell_sorted;
    int *cell_count, *cell_start;   // [ncell_max + 1]
    int *order_tmp, *order;
    int *nlist, *ncount;            // pair rows: nlist[g * 2 kmax + e], g = k / 2; padded with n_atoms to a multiple of 32
    double *blockpart;              // [9 * gridDim.x]
    int *scanpart;                  // [gridDim.x + 1]
    CellGrid *grid;
    double *scal;
    unsigned long long *counters;
    int n_atoms, kmax, max_dim, have_vel, fine_max;
    int zero_pairs;                 // != 0: a density sweep follows; zero counters[kCntPairsInCut] for it
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
    // this kernel precedes every density sweep of new positions: it also zeroes that sweep's pair counter
    if (a.zero_pairs && blockIdx.x == 0 && threadIdx.x == 0) a.counters[kCntPairsInCut] = 0ull;
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
        if (a.xfr) a.xfr[k] = split_record(p);
        a.perm[k] = a.perm_alt[k];
        if (a.have_vel) {
            a.vel[3 * size_t(k)] = a.vel_alt[3 * size_t(k)];
            a.vel[3 * size_t(k) + 1] = a.vel_alt[3 * size_t(k) + 1];
            a.vel[3 * size_t(k) + 2] = a.vel_alt[3 * size_t(k) + 2];
        }
    }
    if (gtid == 0) {                                                             // the dummy records
        a.xs[N] = make_double4(kFarAway, kFarAway, kFarAway, 0.0);
        if (a.xfr) a.xfr[N] = RecF{kFarAwayF, kFarAwayF, kFarAwayF, 0.f, 0.f, 0.f, 0.f, 0.f};
    }
    grid.sync();

    // ---- P8: neighbour rows, one warp per PAIR of consecutive atoms (k0 = 2g, k1 = 2g + 1) ----
    // The row of a pair is the union of the two atoms' neighbourhoods (they sit in the same or in
    // adjacent fine cells, so the union is ~1.2x one neighbourhood): the sweeps fetch every record once
    // for two rows i.  Capacity of a pair row: 2 * kmax entries.
    const double rl2 = a.r_list * a.r_list;
    const double rl2_cells = rl2 * g.inv_edge * g.inv_edge;           // (list radius / edge)^2
    const int G = g.fine;
    // reach[ady][adz]: how many cells along x a neighbour can be away in a row of cells whose nearest points
    // are (ady, adz) cells away in y, z (-1: the row is out of reach)
    __shared__ int reach[kFineMax + 1][kFineMax + 1];
    if (tid < (kFineMax + 1) * (kFineMax + 1)) {
        const int ady = tid / (kFineMax + 1), adz = tid % (kFineMax + 1);
        const double rem = rl2_cells - double(adz * adz + ady * ady);
        reach[ady][adz] = rem > 0.0 ? min(G, int(sqrt(rem)) + 1) : -1;
    }
    __syncthreads();
    const unsigned lt_mask = (1u << lane) - 1u;
    const int cap = 2 * a.kmax;
    int my_max = 0;                                                    // longest single-atom neighbourhood
    bool my_overflow = false;
    const int gwarp = gtid >> 5, nwarps = gsize >> 5;
    const int npairs = (N + 1) >> 1;
    for (int gp = gwarp; gp < npairs; gp += nwarps) {
        const int k0 = 2 * gp, k1 = k0 + 1;
        const bool has1 = k1 < N;
        const double4 p0 = a.xs[k0];
        const double4 p1 = a.xs[has1 ? k1 : N];                        // odd N: the dummy record, never in range
        const int c0 = a.cell_sorted[k0], c1 = has1 ? a.cell_sorted[k1] : c0;
        const int cx0 = c0 % g.nx, cy0 = (c0 / g.nx) % g.ny, cz0 = c0 / (g.nx * g.ny);
        const int cx1 = c1 % g.nx, cy1 = (c1 / g.nx) % g.ny, cz1 = c1 / (g.nx * g.ny);
        int *row = a.nlist + size_t(gp) * cap;
        int cnt = 0, cnt0 = 0, cnt1 = 0;
        // x-range of cells of the row (yy, zz) that can hold a neighbour of an atom in cell (cx, cy, cz)
        auto xrange = [&](int cx, int cy, int cz, int yy, int zz, int &lo, int &hi) -> bool {
            if (abs(zz - cz) > G || abs(yy - cy) > G) return false;
            const int mx = reach[max(abs(yy - cy) - 1, 0)][max(abs(zz - cz) - 1, 0)];
            if (mx < 0) return false;
            lo = max(cx - mx, 0); hi = min(cx + mx, g.nx - 1);
            return true;
        };
        auto scan = [&](int jb, int je) {
            for (int j0 = jb; j0 < je; j0 += 32) {
                const int j = j0 + lane;
                bool in0 = false, in1 = false;
                if (j < je) {
                    const double4 q = a.xs[j];
                    const double ax = p0.x - q.x, ay = p0.y - q.y, az = p0.z - q.z;
                    const double bx = p1.x - q.x, by = p1.y - q.y, bz = p1.z - q.z;
                    in0 = fma(az, az, fma(ay, ay, ax * ax)) < rl2;
                    in1 = fma(bz, bz, fma(by, by, bx * bx)) < rl2;
                }
                const bool ok = in0 || in1;                             // includes k0 and k1 themselves: excluded
                const unsigned m = __ballot_sync(0xffffffffu, ok);      // by index in the sweeps
                const int at = cnt + __popc(m & lt_mask);
                if (ok && at < cap) row[at] = j;
                cnt += __popc(m);
                cnt0 += (in0 && j != k0) ? 1 : 0;                       // per lane; summed over the warp below
                cnt1 += (in1 && j != k1) ? 1 : 0;
            }
        };
        const bool near = abs(cx0 - cx1) <= 2 * G && abs(cy0 - cy1) <= 2 * G && abs(cz0 - cz1) <= 2 * G;
        if (near) {
            // one pass over the bounding box of the two stencils, each row of cells once
            for (int zz = max(min(cz0, cz1) - G, 0); zz <= min(max(cz0, cz1) + G, g.nz - 1); ++zz)
                for (int yy = max(min(cy0, cy1) - G, 0); yy <= min(max(cy0, cy1) + G, g.ny - 1); ++yy) {
                    int lo0, hi0, lo1, hi1;
                    const bool v0 = xrange(cx0, cy0, cz0, yy, zz, lo0, hi0);
                    const bool v1 = has1 && xrange(cx1, cy1, cz1, yy, zz, lo1, hi1);
                    if (!v0 && !v1) continue;
                    const int lo = v0 ? (v1 ? min(lo0, lo1) : lo0) : lo1;
                    const int hi = v0 ? (v1 ? max(hi0, hi1) : hi0) : hi1;
                    const int rowc = (zz * g.ny + yy) * g.nx;
                    scan(a.cell_start[rowc + lo], a.cell_start[rowc + hi + 1]);
                }
        } else {
            // the stencils are disjoint (the pair straddles the end of a row of cells): one pass each
            for (int which = 0; which < 2; ++which) {
                const int cx = which ? cx1 : cx0, cy = which ? cy1 : cy0, cz = which ? cz1 : cz0;
                for (int zz = max(cz - G, 0); zz <= min(cz + G, g.nz - 1); ++zz)
                    for (int yy = max(cy - G, 0); yy <= min(cy + G, g.ny - 1); ++yy) {
                        int lo, hi;
                        if (!xrange(cx, cy, cz, yy, zz, lo, hi)) continue;
                        const int rowc = (zz * g.ny + yy) * g.nx;
                        scan(a.cell_start[rowc + lo], a.cell_start[rowc + hi + 1]);
                    }
            }
        }
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) {
            cnt0 += __shfl_xor_sync(0xffffffffu, cnt0, off);
            cnt1 += __shfl_xor_sync(0xffffffffu, cnt1, off);
        }
        const int kept = min(cnt, cap);
        const int padded = min((kept + 31) & ~31, cap);
        if (kept + lane < padded) row[kept + lane] = N;                 // pad with the dummy record
        if (lane == 0) a.ncount[gp] = kept;
        my_max = max(my_max, max(cnt0, cnt1));
        my_overflow = my_overflow || cnt > cap;
    }
    if (lane == 0 && (my_overflow || my_max > a.kmax)) atomicExch(&a.counters[kCntOverflow], 1ull);
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
    RecF *xfr;                // MIXED: [N + 1] split binary32 records (same order, same dummy); sweep 1 stores fl32(s') here
    const int *nlist;         // [ceil(N/2)][2 * kmax] pair rows, padded with N to a multiple of 32
    const int *ncount;        // [ceil(N/2)]
    int n_atoms, kmax;
    int pairs_per_cta;        // consecutive atom pairs one CTA works through (multiple of warps * 32 / LPA)
    double *rho;              // [N]    sweep 1
    double *force;            // [N*3]  sweep 2
    double *partial;          // [gridDim.x]
    unsigned long long *pairs_in_cut;   // sweep 1: += ordered pairs with r^2 < r_c^2 (zeroed by the host)
    double rc2;
    double shift_m;           // energy-shifted cutoff (SC_OPT_CUTOFF_SHIFT): r_c^-m, taken off every in-range term of sweep 1; else 0
    PairConsts c;
};

constexpr int kNlistMaxBlock = 256;   // threads per CTA of the list sweeps: 32 * warps, chosen by the host

// one 32-byte record with a single 256-bit load (SASS LDG.E.ENL2.256): one L1 wavefront per line touched
__device__ __forceinline__ double4 load_record(const double4 *p) {
    double4 r;
    asm volatile("ld.global.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(r.x), "=d"(r.y), "=d"(r.z), "=d"(r.w) : "l"(p));
    return r;
}

// One row entry against one of the two atoms of the pair: the strict binary64 test r^2 < r_c^2 (reading
// Q7), then the pair terms of the all-pairs sweeps.  `other` is false for the atom's own record (the
// self term is excluded by index).  BRANCH-FREE: an entry that fails the test runs the same
// instructions on r^2 := 1 with its reciprocal (square root) replaced by 0, so every term it adds is an
// exact 0.  (A warp almost never has 32 failing lanes, so a branch would save nothing, and without
// branches the compiler interleaves the 8 independent chains of a batch: 4 entries x 2 atoms.)
// MIXED: pair arithmetic in binary32 on the converted binary64 difference, partial sums in f[]
// (flushed into acc[] by the caller after every batch).
template <int NE, int ME, bool FORCE, bool ENERGY>
__device__ __forceinline__ void nlist_term(const double4 &pi, const double4 &p, bool other, double rc2, double An,
                                           int n_exp, int m_exp, double (&acc)[4], int &npairs) {
    const double dx = pi.x - p.x, dy = pi.y - p.y, dz = pi.z - p.z;
    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    const bool in = (r2 < rc2) && other;
    if constexpr (!FORCE) npairs += in ? 1 : 0;
    {
        const double r2m = in ? r2 : 1.0;
        if constexpr (!FORCE) {
            if constexpr (ME > 0 && ME % 2 == 0) {
                double w = rcp_fast(r2m);
                w = in ? w : 0.0;
                if constexpr (ME == 6) acc[0] = fma(w * w, w, acc[0]);
                else acc[0] += ipow_c<ME / 2>(w);
            } else {
                double y = rsqrt_fast(r2m);
                y = in ? y : 0.0;
                acc[0] += (ME > 0) ? ipow_c<(ME > 0 ? ME : 1)>(y) : ipow_rt(y, m_exp);
            }
        } else {
            double y = rsqrt_fast(r2m);
            y = in ? y : 0.0;
            const double w = y * y;
            const double ss = pi.w + p.w;
            double coef;
            if constexpr (NE == 9 && ME == 6) {
                const double w2 = w * w, w4 = w2 * w2, y3 = w * y;
                coef = w4 * fma(An, y3, -ss);
                if constexpr (ENERGY) acc[3] = fma(w4, y, acc[3]);
            } else {
                const double pm = (ME > 0) ? ipow_c<(ME > 0 ? ME : 1)>(y) : ipow_rt(y, m_exp);
                const double pn = (NE > 0) ? ipow_c<(NE > 0 ? NE : 1)>(y) : ipow_rt(y, n_exp);
                coef = w * fma(An, pn, -ss * pm);
                if constexpr (ENERGY) acc[3] += pn;
            }
            acc[0] = fma(coef, dx, acc[0]);
            acc[1] = fma(coef, dy, acc[1]);
            acc[2] = fma(coef, dz, acc[2]);
        }
    }
}

// MIXED: the same term in binary32 on split records (no binary64 instruction, no conversion on the common path).
// Set membership must equal the oracle's binary64 decision (reading Q7): the binary32 r^2 decides unless it lies
// within 2e-6 r_c^2 of the cutoff (its own error is < 4e-7 relative), in which case the binary64 records are
// fetched and the decision is taken exactly as in the FP64 path.  The hot loop only raises a flag for such an
// entry (~3 in a million); a lane whose flag is up recomputes its share of the row with exact decisions.
struct PairGeomF { float fx, fy, fz, q2; };
__device__ __forceinline__ PairGeomF nlist_geom_f(const RecF &pi, const RecF &p) {
    PairGeomF g;
    g.fx = (pi.xh - p.xh) + (pi.xl - p.xl); g.fy = (pi.yh - p.yh) + (pi.yl - p.yl); g.fz = (pi.zh - p.zh) + (pi.zl - p.zl);
    g.q2 = fmaf(g.fz, g.fz, fmaf(g.fy, g.fy, g.fx * g.fx));
    return g;
}
__device__ __forceinline__ bool nlist_exact_in_range(const double4 *xs, int i, int j, double rc2) {
    const double4 a = xs[i], b = xs[j];
    const double dx = a.x - b.x, dy = a.y - b.y, dz = a.z - b.z;
    return fma(dz, dz, fma(dy, dy, dx * dx)) < rc2;
}
template <int NE, int ME, bool FORCE, bool ENERGY>
__device__ __forceinline__ void nlist_term_f(const RecF &pi, const RecF &p, PairGeomF g, bool in, float Anf, int n_exp,
                                             int m_exp, float (&f)[4], int &npairs) {
    if constexpr (!FORCE) npairs += in ? 1 : 0;
    const float q2 = in ? g.q2 : 1.0f;
    if constexpr (!FORCE) {
        if constexpr (ME > 0 && ME % 2 == 0) {
            float w = rcp_fast_f(q2);
            w = in ? w : 0.f;
            if constexpr (ME == 6) f[0] = fmaf(w * w, w, f[0]);
            else f[0] += ipow_cf<ME / 2>(w);
        } else {
            float y = rsqrt_fast_f(q2);
            y = in ? y : 0.f;
            f[0] += (ME > 0) ? ipow_cf<(ME > 0 ? ME : 1)>(y) : ipow_rtf(y, m_exp);
        }
    } else {
        // a far-away record must not turn 0 * inf into NaN
        const float fx = in ? g.fx : 0.f, fy = in ? g.fy : 0.f, fz = in ? g.fz : 0.f;
        float y = rsqrt_fast_f(q2);
        y = in ? y : 0.f;
        const float w = y * y;
        const float ss = pi.s + p.s;
        float coef;
        if constexpr (NE == 9 && ME == 6) {
            const float w2 = w * w, w4 = w2 * w2, y3 = w * y;
            coef = w4 * fmaf(Anf, y3, -ss);
            if constexpr (ENERGY) f[3] = fmaf(w4, y, f[3]);
        } else {
            const float pm = (ME > 0) ? ipow_cf<(ME > 0 ? ME : 1)>(y) : ipow_rtf(y, m_exp);
            const float pn = (NE > 0) ? ipow_cf<(NE > 0 ? NE : 1)>(y) : ipow_rtf(y, n_exp);
            coef = w * fmaf(Anf, pn, -ss * pm);
            if constexpr (ENERGY) f[3] += pn;
        }
        f[0] = fmaf(coef, fx, f[0]);
        f[1] = fmaf(coef, fy, f[1]);
        f[2] = fmaf(coef, fz, f[2]);
    }
}

// LPA lanes per atom PAIR (32 / LPA pairs per warp at a time).  A CTA works through pairs_per_cta
// consecutive pairs of the internal (cell) order, its warps interleaved, so that the records its
// gathers touch stay in L1.  Every fetched record serves both atoms of the pair.
// SHIFT (sweep 1 only): energy-shifted cutoff -- the in-range entries are counted per atom and the epilogue takes
// count * r_c^-m off the sum (a separate instantiation: the per-atom counters cost the plain sweep 5 %).
template <int LPA, int NE, int ME, bool FORCE, bool ENERGY, bool MIXED, bool SHIFT = false>
__global__ void __launch_bounds__(kNlistMaxBlock) nlist_kernel(const NlistArgs a) {
    constexpr int AW = 32 / LPA;                         // pairs per warp
    __shared__ double scratch[32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int g = lane / LPA, q = lane % LPA;            // group g of the warp takes one pair, q strides its row
    const int N = a.n_atoms, NP = (N + 1) >> 1;
    const int n_exp = (NE > 0) ? NE : a.c.n, m_exp = (ME > 0) ? ME : a.c.m;
    const double An = a.c.An, rc2 = a.rc2;
    const float Anf = float(An), rc2f = float(rc2), band = 2.0e-6f * rc2f;
    const size_t stride = 2 * size_t(a.kmax);
    double contrib = 0.0;
    int npairs = 0;

    const int base = blockIdx.x * a.pairs_per_cta;
    const int end = min(NP, base + a.pairs_per_cta);
    const int nwarps = blockDim.x >> 5;
    for (int g0 = base + warp * AW; g0 < end; g0 += nwarps * AW) {
        const int gp = g0 + g;
        const bool live = gp < end;
        const int i0 = live ? 2 * gp : N, i1 = (live && 2 * gp + 1 < N) ? 2 * gp + 1 : N;   // N = the dummy record
        // records: binary64 (x, y, z, s') or, MIXED, their split binary32 twins -- both 32 bytes, fetched alike
        const double4 *recs = MIXED ? reinterpret_cast<const double4 *>(a.xfr) : a.xs;
        const double4 pa = recs[i0], pb = recs[i1];
        const int cnt = live ? a.ncount[gp] : 0;
        const int niter = (cnt + LPA - 1) / LPA;         // rows are padded to a multiple of 32 >= LPA
        const int *row = a.nlist + size_t(live ? gp : 0) * stride + q;
        double acc0[4] = {0.0, 0.0, 0.0, 0.0}, acc1[4] = {0.0, 0.0, 0.0, 0.0};
        float f0[4] = {0.f, 0.f, 0.f, 0.f}, f1[4] = {0.f, 0.f, 0.f, 0.f};
        int np0 = 0, np1 = 0;                            // sweep 1: in-range entries (SHIFT: of each atom of the pair)
        bool unsure = false;

        auto entry = [&](int j, const double4 &p) {
            if constexpr (MIXED) {
                // binary32 decision; entries too close to the cutoff to trust it only raise `unsure`
                const RecF &fa = reinterpret_cast<const RecF &>(pa), &fb = reinterpret_cast<const RecF &>(pb);
                const RecF &fp = reinterpret_cast<const RecF &>(p);
                const PairGeomF ga = nlist_geom_f(fa, fp), gb = nlist_geom_f(fb, fp);
                unsure = unsure || fabsf(ga.q2 - rc2f) <= band || fabsf(gb.q2 - rc2f) <= band;
                nlist_term_f<NE, ME, FORCE, ENERGY>(fa, fp, ga, ga.q2 < rc2f && j != i0, Anf, n_exp, m_exp, f0, np0);
                nlist_term_f<NE, ME, FORCE, ENERGY>(fb, fp, gb, gb.q2 < rc2f && j != i1, Anf, n_exp, m_exp, f1, SHIFT ? np1 : np0);
            } else {
                nlist_term<NE, ME, FORCE, ENERGY>(pa, p, j != i0, rc2, An, n_exp, m_exp, acc0, np0);
                nlist_term<NE, ME, FORCE, ENERGY>(pb, p, j != i1, rc2, An, n_exp, m_exp, acc1, SHIFT ? np1 : np0);
            }
        };
        auto flush = [&]() {
            if constexpr (MIXED) {
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    acc0[c] += double(f0[c]); acc1[c] += double(f1[c]);
                    f0[c] = 0.f; f1[c] = 0.f;
                }
            }
        };
        // Software pipeline over batches of CH entries per lane: while batch t is in the FP64 pipe the
        // records of batch t + 1 (indices fetched an iteration earlier) and the indices of batch t + 2
        // (streamed from HBM) are in flight.  Slots beyond the row read the dummy record.
        constexpr int CH = 4;
        const int nbatch = (niter + CH - 1) / CH;
        auto load_idx = [&](int b, int (&jj)[CH]) {
#pragma unroll
            for (int u = 0; u < CH; ++u) {
                const int it = b * CH + u;
                jj[u] = it < niter ? row[it * LPA] : N;
            }
        };
        int jc[CH], j1[CH], j2[CH];
        double4 pc[CH], pn[CH];
        load_idx(0, jc);
        load_idx(1, j1);
#pragma unroll
        for (int u = 0; u < CH; ++u) pc[u] = load_record(recs + jc[u]);
        for (int b = 0; b < nbatch; ++b) {
            load_idx(b + 2, j2);
#pragma unroll
            for (int u = 0; u < CH; ++u) pn[u] = load_record(recs + j1[u]);
#pragma unroll
            for (int u = 0; u < CH; ++u) entry(jc[u], pc[u]);
            flush();
#pragma unroll
            for (int u = 0; u < CH; ++u) { jc[u] = j1[u]; j1[u] = j2[u]; pc[u] = pn[u]; }
        }

        if constexpr (MIXED) {
            if (unsure) {
                // Rare (~3 entries in a million): this lane met an entry whose binary32 r^2 is within 2e-6 r_c^2 of the
                // cutoff.  Its partial sums are recomputed with every decision taken from the binary64 records, exactly
                // as the FP64 path takes it (reading Q7: set membership is the oracle's).
#pragma unroll
                for (int c = 0; c < 4; ++c) { acc0[c] = 0.0; acc1[c] = 0.0; f0[c] = 0.f; f1[c] = 0.f; }
                np0 = 0; np1 = 0;
                const RecF &fa = reinterpret_cast<const RecF &>(pa), &fb = reinterpret_cast<const RecF &>(pb);
                for (int it = 0; it < niter; ++it) {
                    const int j = row[it * LPA];
                    const double4 p = load_record(recs + j);
                    const RecF &fp = reinterpret_cast<const RecF &>(p);
                    const bool in0 = j != i0 && nlist_exact_in_range(a.xs, i0, j, rc2);
                    const bool in1 = j != i1 && nlist_exact_in_range(a.xs, i1, j, rc2);
                    nlist_term_f<NE, ME, FORCE, ENERGY>(fa, fp, nlist_geom_f(fa, fp), in0, Anf, n_exp, m_exp, f0, np0);
                    nlist_term_f<NE, ME, FORCE, ENERGY>(fb, fp, nlist_geom_f(fb, fp), in1, Anf, n_exp, m_exp, f1, SHIFT ? np1 : np0);
                    if ((it & 3) == 3) flush();                  // same flush points as the fast loop
                }
                flush();
            }
        }
        npairs += np0 + np1;
        if constexpr (!FORCE && SHIFT) {
            // per-atom neighbour counts over the LPA lanes (integers: exact), for the shifted density
#pragma unroll
            for (int off = LPA / 2; off > 0; off >>= 1) {
                np0 += __shfl_xor_sync(0xffffffffu, np0, off);
                np1 += __shfl_xor_sync(0xffffffffu, np1, off);
            }
        }

        // ---- reduce over the LPA lanes of the pair (fixed order) ----
        constexpr int NV = FORCE ? (ENERGY ? 4 : 3) : 1;
#pragma unroll
        for (int c = 0; c < NV; ++c) { acc0[c] = group_sum<LPA>(acc0[c]); acc1[c] = group_sum<LPA>(acc1[c]); }
        if (live && q == 0) {
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int i = h ? i1 : i0;
                const double *acc = h ? acc1 : acc0;
                if (i >= N) continue;
                if constexpr (!FORCE) {
                    // shifted cutoff: every in-range term loses r_c^-m
                    const double rho = SHIFT ? a.c.am * fma(-double(h ? np1 : np0), a.shift_m, acc[0]) : a.c.am * acc[0];
                    a.rho[i] = rho;
                    const double root = rho > 0.0 ? sqrt(rho) : 0.0;       // reading Q9
                    const double sp = rho > 0.0 ? a.c.Bm / root : 0.0;
                    a.xs[i].w = sp;
                    if constexpr (MIXED) a.xfr[i].s = float(sp);
                    contrib += root;
                } else {
                    a.force[3 * size_t(i)] = acc[0];
                    a.force[3 * size_t(i) + 1] = acc[1];
                    a.force[3 * size_t(i) + 2] = acc[2];
                    contrib += acc[3];
                }
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
// new positions, a new row capacity or a new cell size: the rows are rebuilt at the next evaluation, and an overflow
// recorded for the old ones says nothing about the new ones
__global__ void reset_list_state_kernel(unsigned long long *__restrict__ counters, double *__restrict__ scal) {
    counters[kCntListValid] = 0ull;
    counters[kCntOverflow] = 0ull;
    scal[kSlotMaxDisp2] = 0.0;
}
__global__ void zero_u64_kernel(unsigned long long *p) { *p = 0ull; }
#endif  // SCMD_MAIN_TU

}  // namespace scmd
