// sc_cutoff.cuh -- the cutoff variant (BASELINE.json; the paper itself runs all pairs and names
// cutoffs as work in progress): cell binning by counting sort, Verlet neighbour
// rows with a skin, and the two list-driven sweeps.
//
// Design constraints (measured, profiles/ncu_cutoff_r1.md, profiles/ncu_cutoff_r2.md): a list-driven FP64 sweep on
// sm_100a is bound by the FP64 pipe only if (i) the 32 lanes of a warp gather ADJACENT records (one L1 wavefront
// per distinct 128-byte line), (ii) every fetched record is used for more than one row i, and (iii) the index
// stream does not come from DRAM one 4-byte entry per pair (round 1: 78 MB per sweep at N = 65536, 25x the
// algorithmic bytes, and a dependent DRAM -> L2 load chain in the hot loop).  Hence:
//   * atoms are sorted into FINE cells (edge = list radius / G, G = 4 by default), x fastest, so the
//     in-range neighbours of an atom are ~60 contiguous runs of the internal order;
//   * a neighbour row belongs to a PAIR of consecutive atoms (the union of their neighbourhoods, ~1.2x one
//     of them) and is stored RUN-LENGTH encoded: one 32-bit word (first index << 5 | length - 1) per run of
//     up to 32 consecutive atoms -- ~70-90 words instead of ~560 entries per row (N = 65536: ~10 MB instead
//     of 74 MB, L2-resident);
//   * one WARP walks one row: it expands the runs into a shared-memory index list (a warp scan and a few
//     stores per 32 runs), then works through it in dense batches of 32 entries, lane t taking entry
//     32 b + t: adjacent lanes gather adjacent records with one 256-bit load each (SASS LDG.E.ENL2.256) and
//     evaluate them against both atoms of the pair; the index stream never touches DRAM in the loop.
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
//   P8  neighbour rows, one warp per atom pair: the <= (2G+1)^2 rows of cells in (y, z) that can hold a
//       neighbour each contribute ONE contiguous index range; the ranges are computed 32 at a time (one per
//       lane, all cell_start loads in flight together), expanded into a shared-memory candidate list and
//       tested in dense batches of 32 candidates; every j within r_c + skin of EITHER atom goes into the row,
//       as runs (ballot + bit scans); rows never truncate silently (overflow flag -> SC_ERR_CAPACITY)
// After a build the library's internal atom order IS the cell order; perm[k] = caller's index.
//
// nlist_kernel: applies the strict binary64 test r^2 < r_c^2 (reading Q7: same decision value as the oracle) to
// every entry and accumulates the same pair terms as the all-pairs sweeps.  MIXED: the rows gather split binary32
// records (x = xh + xl) and the whole pair term runs in binary32 -- no conversion, no binary64 instruction -- except
// that an entry whose binary32 r^2 lies within 2e-6 r_c^2 of the cutoff takes its set-membership decision from the
// binary64 records (reading Q7: membership is the oracle's, bit for bit); partial sums are flushed into binary64
// after every batch.
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

constexpr bool kListRuns = true;  // rows as run-length words (true) or as one 32-bit index per entry (false): measured, DESIGN.md 6.3
constexpr int kRunBits = 3;      // a run word = first index << kRunBits | (length - 1): runs of 1 .. 8 atoms (short runs keep
                                 // the expansion loop of the sweeps short: every lane writes out one run)
constexpr int kRunMaxLen = 1 << kRunBits;
constexpr int64_t kCutoffMaxAtoms = int64_t(1) << (32 - kRunBits);   // first index must fit in 29 bits
constexpr int kCandCap = 1024;   // rebuild P8: candidates expanded per chunk of 32 cell-row ranges, per warp
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
    int *nlist, *ncount;            // pair rows g = k / 2: nlist[g * 2 kmax + r] = run r (start << 5 | len - 1), ncount[g] runs
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
        // the 9 quantities over all CTAs' partials: 28 threads per quantity stride the CTAs, then one thread per quantity
        // combines the 28 in a fixed order (one thread walking all CTAs took 91 us of a 330 us build at N = 65536)
        __shared__ double comb[9][28];
        if (tid < 9 * 28) {
            const int q = tid / 28, r = tid % 28;
            double v = q < 3 ? 0.0 : (q < 6 ? 1e300 : -1e300);
            for (int b = r; b < int(gridDim.x); b += 28) {
                const double o = a.blockpart[9 * b + q];
                v = q < 3 ? v + o : (q < 6 ? fmin(v, o) : fmax(v, o));
            }
            comb[q][r] = v;
        }
        __syncthreads();
        if (tid < 9) {
            double v = comb[tid][0];
            for (int r = 1; r < 28; ++r) v = tid < 3 ? v + comb[tid][r] : (tid < 6 ? fmin(v, comb[tid][r]) : fmax(v, comb[tid][r]));
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
    // for two rows i.  Stored as runs of consecutive indices; capacity of a pair row: 2 * kmax words.
    const double rl2 = a.r_list * a.r_list;
    const double rl2_cells = rl2 * g.inv_edge * g.inv_edge;           // (list radius / edge)^2
    const int G = g.fine;
    // reach[ady][adz]: how many cells along x a neighbour can be away in a row of cells whose nearest points
    // are (ady, adz) cells away in y, z (-1: the row is out of reach)
    __shared__ int reach[kFineMax + 1][kFineMax + 1];
    __shared__ int cand_all[8][kCandCap];
    int *cand = cand_all[warp];
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
        // the row holds neither k0 nor k1: the sweeps add the term between the two themselves, in a free lane of the
        // row's last batch, so no entry is ever an atom's own record and no sweep compares indices (the self term is
        // excluded by index, reading Q11 -- here, once, at the build)
        int nruns = 0, cnt0 = 0, cnt1 = 0;
        // x-range of cells of the row (yy, zz) that can hold a neighbour of an atom in cell (cx, cy, cz)
        auto xrange = [&](int cx, int cy, int cz, int yy, int zz, int &lo, int &hi) -> bool {
            if (abs(zz - cz) > G || abs(yy - cy) > G) return false;
            const int mx = reach[max(abs(yy - cy) - 1, 0)][max(abs(zz - cz) - 1, 0)];
            if (mx < 0) return false;
            lo = max(cx - mx, 0); hi = min(cx + mx, g.nx - 1);
            return true;
        };
        // 32 candidates (consecutive entries of the candidate list; `valid` lanes only): distance tests against
        // both atoms, then the accepted ones are appended to the row as runs of consecutive indices (never across a
        // batch, never longer than kRunMaxLen).
        auto batch = [&](int j, bool valid) {
            bool in0 = false, in1 = false;
            if (valid) {
                const double4 q = a.xs[j];
                const double ax = p0.x - q.x, ay = p0.y - q.y, az = p0.z - q.z;
                const double bx = p1.x - q.x, by = p1.y - q.y, bz = p1.z - q.z;
                in0 = fma(az, az, fma(ay, ay, ax * ax)) < rl2;
                in1 = fma(bz, bz, fma(by, by, bx * bx)) < rl2;
            }
            const bool ok = (in0 || in1) && j != k0 && j != k1;         // never the pair itself (see above)
            const int pj = __shfl_up_sync(0xffffffffu, j, 1);
            const int pok = __shfl_up_sync(0xffffffffu, ok ? 1 : 0, 1);
            const bool fresh = ok && (lane == 0 || !pok || pj != j - 1);       // a run of consecutive indices begins here
            const unsigned fm = __ballot_sync(0xffffffffu, fresh);
            // runs are cut after kRunMaxLen entries: position inside the run = lane - (last `fresh` lane at or before it)
            const int since = lane - (31 - __clz(int(fm & (0xffffffffu >> (31 - lane)))));
            const bool start = ok && (fresh || (since & (kRunMaxLen - 1)) == 0);
            const unsigned s = __ballot_sync(0xffffffffu, start), o = __ballot_sync(0xffffffffu, ok);
            if constexpr (kListRuns) {
                if (start) {
                    const unsigned cont = o & ~s;                        // lanes that continue the run of the lane before
                    const unsigned x = lane == 31 ? 0u : (cont >> (lane + 1));
                    const int len = __ffs(int(~x));                      // 1 + number of continuation lanes that follow
                    const int at = nruns + __popc(s & lt_mask);
                    if (at < cap) row[at] = int((unsigned(j) << kRunBits) | unsigned(len - 1));
                }
                nruns += __popc(s);
            } else {
                const int at = nruns + __popc(o & lt_mask);              // one word per entry, ascending
                if (ok && at < cap) row[at] = j;
                nruns += __popc(o);
            }
            cnt0 += (in0 && j != k0) ? 1 : 0;                            // per lane; summed over the warp below
            cnt1 += (in1 && j != k1) ? 1 : 0;
        };
        // one contiguous index range per row of cells; ranges are computed 32 at a time (one per lane), expanded
        // into the candidate list of this warp and tested in dense batches
        auto sweep_box = [&](int ylo, int yhi, int zlo, int zhi, int which) {
            const int nyb = yhi - ylo + 1, R = nyb * (zhi - zlo + 1);
            for (int r0 = 0; r0 < R; r0 += 32) {
                const int r = r0 + lane;
                int jb = 0, len = 0;
                if (r < R) {
                    const int zz = zlo + r / nyb, yy = ylo + r % nyb;
                    int lo0 = 0, hi0 = -1, lo1 = 0, hi1 = -1;
                    const bool v0 = which != 1 && xrange(cx0, cy0, cz0, yy, zz, lo0, hi0);
                    const bool v1 = which != 0 && has1 && xrange(cx1, cy1, cz1, yy, zz, lo1, hi1);
                    if (v0 || v1) {
                        const int lo = v0 ? (v1 ? min(lo0, lo1) : lo0) : lo1;
                        const int hi = v0 ? (v1 ? max(hi0, hi1) : hi0) : hi1;
                        const int rowc = (zz * g.ny + yy) * g.nx;
                        jb = a.cell_start[rowc + lo];
                        len = a.cell_start[rowc + hi + 1] - jb;
                    }
                }
                int incl = len;
#pragma unroll
                for (int off = 1; off < 32; off <<= 1) {
                    const int v = __shfl_up_sync(0xffffffffu, incl, off);
                    if (lane >= off) incl += v;
                }
                const int total = __shfl_sync(0xffffffffu, incl, 31);
                if (total == 0) continue;
                if (total <= kCandCap) {
                    int longest = len;
#pragma unroll
                    for (int off = 16; off > 0; off >>= 1) longest = max(longest, __shfl_xor_sync(0xffffffffu, longest, off));
                    const int base = incl - len;
                    for (int k = 0; k < longest; ++k)
                        if (k < len) cand[base + k] = jb + k;
                    __syncwarp();
                    for (int q0 = 0; q0 < total; q0 += 32) {
                        const int q = q0 + lane;
                        const bool valid = q < total;
                        batch(valid ? cand[q] : 0, valid);
                    }
                    __syncwarp();
                } else {
                    // very long ranges (clamped boundary cells, compressed matter): range by range
                    for (int rr = 0; rr < 32; ++rr) {
                        const int jb_r = __shfl_sync(0xffffffffu, jb, rr), len_r = __shfl_sync(0xffffffffu, len, rr);
                        for (int t0 = 0; t0 < len_r; t0 += 32) batch(jb_r + t0 + lane, t0 + lane < len_r);
                    }
                }
            }
        };
        const bool near = abs(cx0 - cx1) <= 2 * G && abs(cy0 - cy1) <= 2 * G && abs(cz0 - cz1) <= 2 * G;
        if (near) {
            // one pass over the bounding box of the two stencils, each row of cells once
            sweep_box(max(min(cy0, cy1) - G, 0), min(max(cy0, cy1) + G, g.ny - 1), max(min(cz0, cz1) - G, 0),
                      min(max(cz0, cz1) + G, g.nz - 1), 2);
        } else {
            // the stencils are disjoint (the pair straddles the end of a row of cells): one pass each
            sweep_box(max(cy0 - G, 0), min(cy0 + G, g.ny - 1), max(cz0 - G, 0), min(cz0 + G, g.nz - 1), 0);
            if (has1) sweep_box(max(cy1 - G, 0), min(cy1 + G, g.ny - 1), max(cz1 - G, 0), min(cz1 + G, g.nz - 1), 1);
        }
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) {
            cnt0 += __shfl_xor_sync(0xffffffffu, cnt0, off);
            cnt1 += __shfl_xor_sync(0xffffffffu, cnt1, off);
        }
        if constexpr (!kListRuns) {
            // one free slot for the term between the two atoms of the pair, then the dummy record up to a whole batch
            const int padded = min((nruns + 32) & ~31, cap);
            if (nruns + lane < padded) row[nruns + lane] = N;
            my_overflow = my_overflow || nruns + 1 > cap;
        }
        if (lane == 0) a.ncount[gp] = min(nruns, cap);
        my_max = max(my_max, max(cnt0, cnt1));
        my_overflow = my_overflow || nruns > cap;
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
    const int *nlist;         // [ceil(N/2)][2 * kmax] pair rows of run words (first index << 5 | length - 1)
    const int *ncount;        // [ceil(N/2)] runs per row
    int n_atoms, kmax;
    int pairs_per_cta;        // consecutive atom pairs in one block of rows (a multiple of the warps per CTA); CTA c takes
                              //   the blocks c, c + gridDim.x, ...
    int idx_cap;              // ints of shared memory per warp for the expanded row: >= 2 kmax + 64
    double *rho;              // [N]    sweep 1
    double *force;            // [N*3]  sweep 2
    double *partial;          // [gridDim.x]
    unsigned long long *pairs_in_cut;   // sweep 1: += ordered pairs with r^2 < r_c^2 (zeroed by the host)
    double rc2;
    double shift_m;           // energy-shifted cutoff (SC_OPT_CUTOFF_SHIFT): r_c^-m, taken off every in-range term of sweep 1; else 0
    PairConsts c;
};

constexpr int kNlistMaxBlock = 128;   // threads per CTA of the list sweeps: 32 * warps (<= 4), chosen by the host
constexpr int kNlistMinBlocks = 6;    // resident CTAs per SM the register allocation must allow (<= 85 registers)

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

// The same terms for entries that cannot be the atom itself (every batch but the first of a row): no index compare,
// and ONE select per term instead of five -- the MUFU seed of the reciprocal (square root) comes with a zero low word,
// so an entry that fails the test gets the seed's high word replaced by 0 and every later product is an exact 0
// (r^2 of two different atoms is a positive finite number: no 0 x inf on the way; the dummy record gives r^2 = 3e300).
__device__ __forceinline__ double seed_or_zero(double seed, bool keep) {
    return __hiloint2double(keep ? __double2hiint(seed) : 0, 0);
}
template <int NE, int ME, bool FORCE, bool ENERGY>
__device__ __forceinline__ void nlist_term_lean(const double4 &pi, const double4 &p, double rc2, double An, int n_exp,
                                                int m_exp, double (&acc)[4], int &npairs) {
    const double dx = pi.x - p.x, dy = pi.y - p.y, dz = pi.z - p.z;
    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    const bool in = r2 < rc2;
    if constexpr (!FORCE) {
        npairs += in ? 1 : 0;
        if constexpr (ME > 0 && ME % 2 == 0) {
            const double y0 = seed_or_zero(rcp_seed(r2), in);
            const double e = fma(-r2, y0, 1.0);
            const double w = fma(y0, fma(e, e, e), y0);
            if constexpr (ME == 6) acc[0] = fma(w * w, w, acc[0]);
            else acc[0] += ipow_c<ME / 2>(w);
        } else {
            const double y0 = seed_or_zero(rsqrt_seed(r2), in);
            const double t = r2 * y0, e = fma(-t, y0, 1.0);
            const double y = fma(y0, e * fma(0.375, e, 0.5), y0);
            acc[0] += (ME > 0) ? ipow_c<(ME > 0 ? ME : 1)>(y) : ipow_rt(y, m_exp);
        }
    } else {
        const double y0 = seed_or_zero(rsqrt_seed(r2), in);
        const double t = r2 * y0, e = fma(-t, y0, 1.0);
        const double y = fma(y0, e * fma(0.375, e, 0.5), y0);
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
template <int NE, int ME, bool FORCE, bool ENERGY>
__device__ __forceinline__ void nlist_term_f_lean(const RecF &pi, const RecF &p, PairGeomF g, bool in, float Anf, int n_exp,
                                                  int m_exp, float (&f)[4], int &npairs) {
    // binary32: g.q2 of the dummy record is 3e36 (finite), of two different atoms > 0
    if constexpr (!FORCE) {
        npairs += in ? 1 : 0;
        if constexpr (ME > 0 && ME % 2 == 0) {
            float y0;
            asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y0) : "f"(g.q2));
            y0 = in ? y0 : 0.f;
            const float w = fmaf(y0, fmaf(-g.q2, y0, 1.0f), y0);
            if constexpr (ME == 6) f[0] = fmaf(w * w, w, f[0]);
            else f[0] += ipow_cf<ME / 2>(w);
        } else {
            float y0;
            asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y0) : "f"(g.q2));
            y0 = in ? y0 : 0.f;
            const float y = fmaf(y0 * fmaf(-(g.q2 * y0), y0, 1.0f), 0.5f, y0);
            f[0] += (ME > 0) ? ipow_cf<(ME > 0 ? ME : 1)>(y) : ipow_rtf(y, m_exp);
        }
    } else {
        float y0;
        asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y0) : "f"(g.q2));
        y0 = in ? y0 : 0.f;
        const float y = fmaf(y0 * fmaf(-(g.q2 * y0), y0, 1.0f), 0.5f, y0);
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
        f[0] = fmaf(coef, g.fx, f[0]);
        f[1] = fmaf(coef, g.fy, f[1]);
        f[2] = fmaf(coef, g.fz, f[2]);
    }
}

// One warp per atom PAIR.  A CTA works through pairs_per_cta consecutive pairs of the internal (cell) order, its
// warps interleaved, so that the records its gathers touch stay in L1.
//
// Row walk.  The run words of a row arrive in registers one row AHEAD (fetched while the row before is in the FP64
// pipe: the list never stalls the loop on DRAM).  The warp expands them into its shared-memory index list -- a warp
// scan of the lengths, then every lane writes out its run of <= 8 indices -- pads the last batch with the index of
// the dummy record and works through the list in batches of 32 entries, lane t taking entry 32 b + t: adjacent
// lanes gather adjacent records with one 256-bit load each (SASS LDG.E.ENL2.256), and every fetched record serves
// both atoms of the pair.  The rows hold no atom's own record (the build excludes the pair itself), so no term
// compares indices; the term BETWEEN the two atoms of the pair rides in the first free lane of the last batch, whose
// "record" is the other atom of the pair.  Issue slots matter as much as the FP64 pipe here (round 1: 101 instructions
// per batch for 46 FP64 ones; now ~57): one select per term, no compares, no register moves.
// SHIFT (sweep 1 only): energy-shifted cutoff -- the in-range entries are counted per atom and the epilogue takes
// count * r_c^-m off the sum (a separate instantiation: the per-atom counters cost the plain sweep 5 %).
constexpr int kNlistCH = 4;           // batches of 32 entries per loop iteration: 2 kNlistCH independent chains per lane
constexpr bool kNlistPF = false;      // records of iteration t + 1 in flight (registers) while iteration t is in the pipe
constexpr int kNlistL1PF = 0;         // records of iteration t + kNlistL1PF are prefetched into L1 (0: off)
constexpr int kNlistRW = 4;           // run words per lane fetched a row ahead (rows of up to 128 runs: fcc rows have ~100)

__device__ __forceinline__ void prefetch_l1(const void *p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }

// sum of V values over the 32 lanes in V / 2 + V / 4 + ... + 1 + (remaining stages) shuffles instead of 5 V: at every
// halving stage a lane keeps one half of its values and hands the other half to its partner.  On return v[0] of lane L
// holds the total of value number L / (32 / V); fixed order, same bits every run.
template <int V>
__device__ __forceinline__ void transpose_sum(double (&v)[V]) {
    const int lane = threadIdx.x & 31;
    int off = 16;
#pragma unroll
    for (int n = V; n > 1; n >>= 1, off >>= 1) {
        const bool upper = (lane & off) != 0;
#pragma unroll
        for (int k = 0; k < n / 2; ++k) {
            const double keep = upper ? v[n / 2 + k] : v[k], give = upper ? v[k] : v[n / 2 + k];
            v[k] = keep + __shfl_xor_sync(0xffffffffu, give, off);
        }
    }
    for (; off > 0; off >>= 1) v[0] += __shfl_xor_sync(0xffffffffu, v[0], off);
}

template <int NE, int ME, bool FORCE, bool ENERGY, bool MIXED, bool SHIFT = false>
__global__ void __launch_bounds__(kNlistMaxBlock, kNlistMinBlocks) nlist_kernel(const NlistArgs a) {
    constexpr int CH = kNlistCH, RW = kNlistRW;
    extern __shared__ int idx_all[];
    __shared__ double scratch[32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int *idx = idx_all + size_t(warp) * a.idx_cap;
    const int N = a.n_atoms, NP = (N + 1) >> 1;
    const int n_exp = (NE > 0) ? NE : a.c.n, m_exp = (ME > 0) ? ME : a.c.m;
    const double An = a.c.An, rc2 = a.rc2;
    const float Anf = float(An), rc2f = float(rc2), band = 2.0e-6f * rc2f;
    const size_t stride = 2 * size_t(a.kmax);
    double contrib = 0.0;
    int npairs = 0;
    // records: binary64 (x, y, z, s') or, MIXED, their split binary32 twins -- both 32 bytes, fetched alike
    const double4 *recs = MIXED ? reinterpret_cast<const double4 *>(a.xfr) : a.xs;

    // Persistent CTAs: the grid is one wave; CTA c works through the blocks c, c + gridDim.x, ... of pairs_per_cta
    // consecutive pairs (static, so every sum keeps a fixed order; strided, so surface and bulk rows mix in every CTA).
    const int nwarps = blockDim.x >> 5;
    const int ppc = a.pairs_per_cta;
    const int cap = int(stride);
    const int lim = 2 * a.kmax + 32;         // a row that passed the capacity check expands to <= 2 kmax entries; one that
                                             // did not (SC_ERR_CAPACITY is on its way) is cut here: no write beyond idx_cap
    auto next_row = [&](int g) {             // the row this warp takes after row g
        const int n = g + nwarps;
        return (n % ppc) < nwarps && n % ppc == warp ? n + (int(gridDim.x) - 1) * ppc : n;
    };
    int nr = 0;
    unsigned rw[RW];
    auto fetch_row = [&](int g, int &n_runs, unsigned (&w)[RW]) {
        if (g < NP) {
            n_runs = a.ncount[g];
            const int *rp = a.nlist + size_t(g) * stride;
#pragma unroll
            for (int u = 0; u < RW; ++u) w[u] = (u * 32 + lane < cap) ? unsigned(rp[u * 32 + lane]) : 0u;
            if (lane < 2 && 2 * g + lane < N) prefetch_l1(recs + 2 * g + lane);   // the two atoms of that pair
        }
    };
    fetch_row(blockIdx.x * ppc + warp, nr, rw);
    for (int gp = blockIdx.x * ppc + warp; gp < NP; gp = next_row(gp)) {
        const int i0 = 2 * gp, i1 = (2 * gp + 1 < N) ? 2 * gp + 1 : N;      // N = the dummy record
        const double4 pa = recs[i0];
        double4 pb = recs[i1];
        if (i1 == N) {
            // odd N: the last pair has a phantom second atom.  It must be far from every atom AND from the dummy record
            // that pads the batches (no term compares indices): the dummy mirrored through the origin
            if constexpr (MIXED) {
                RecF ph{-kFarAwayF, -kFarAwayF, -kFarAwayF, 0.f, 0.f, 0.f, 0.f, 0.f};
                pb = reinterpret_cast<const double4 &>(ph);
            } else {
                pb = make_double4(-kFarAway, -kFarAway, -kFarAway, 0.0);
            }
        }
        const int *rowp = a.nlist + size_t(gp) * stride;
        int nr_next = 0;
        unsigned rw_next[RW];
        fetch_row(next_row(gp), nr_next, rw_next);
        nr = __shfl_sync(0xffffffffu, nr, 0);                                // the same in every lane: say so

        int fill = 0;
        const int *list;                                                     // the row's entries, one index per word
      if constexpr (kListRuns) {
        // ---- expand the runs ----
        __syncwarp();                                                        // the previous row's readers are done
        auto expand = [&](unsigned run, bool live) {
            int len = live ? int(run & (kRunMaxLen - 1)) + 1 : 0;
            const int first = int(run >> kRunBits);
            int incl = len;
#pragma unroll
            for (int off = 1; off < 32; off <<= 1) {
                const int v = __shfl_up_sync(0xffffffffu, incl, off);
                if (lane >= off) incl += v;
            }
            const int at = fill + incl - len;
            len = min(len, max(lim - at, 0));
            int *dst = idx + at;
#pragma unroll
            for (int k = 0; k < kRunMaxLen; ++k)
                if (k < len) dst[k] = first + k;
            fill = min(fill + __shfl_sync(0xffffffffu, incl, 31), lim);
        };
#pragma unroll
        for (int u = 0; u < RW; ++u)
            if (u * 32 < nr) expand(rw[u], u * 32 + lane < nr);
        for (int r0 = RW * 32; r0 < nr; r0 += 32)                            // rows longer than the prefetched part
            expand(r0 + lane < nr ? unsigned(rowp[r0 + lane]) : 0u, r0 + lane < nr);
        // the last batch: entries, then ONE lane for the term between the two atoms of the pair, then the dummy record
        if (lane >= (fill & 31)) idx[fill - (fill & 31) + lane] = N;
        __syncwarp();
        list = idx;
      } else {
        fill = min(nr, cap - 1);                                             // the build padded the row the same way
        list = rowp;
      }
        const int lpair = fill & 31;
        const int nb32 = (fill >> 5) + 1, nwhole = (nb32 - 1) / CH;          // nwhole iterations of CH batches, then 1 .. CH batches

        double acc0[4] = {0.0, 0.0, 0.0, 0.0}, acc1[4] = {0.0, 0.0, 0.0, 0.0};
        float f0[4] = {0.f, 0.f, 0.f, 0.f}, f1[4] = {0.f, 0.f, 0.f, 0.f};
        int np0 = 0, np1 = 0;                            // sweep 1: in-range entries (SHIFT: of each atom of the pair)
        bool unsure = false;

        // one fetched record against both atoms of the pair (qa = qb = the record), or -- the pair lane of the last
        // batch -- each atom against the other (qa = pb, qb = pa)
        auto entry2 = [&](const double4 &qa, const double4 &qb) {
            if constexpr (MIXED) {
                // binary32 decision; entries too close to the cutoff to trust it only raise `unsure`
                const RecF &fa = reinterpret_cast<const RecF &>(pa), &fb = reinterpret_cast<const RecF &>(pb);
                const RecF &ga_ = reinterpret_cast<const RecF &>(qa), &gb_ = reinterpret_cast<const RecF &>(qb);
                const PairGeomF ga = nlist_geom_f(fa, ga_), gb = nlist_geom_f(fb, gb_);
                unsure = unsure || fabsf(ga.q2 - rc2f) <= band || fabsf(gb.q2 - rc2f) <= band;
                nlist_term_f_lean<NE, ME, FORCE, ENERGY>(fa, ga_, ga, ga.q2 < rc2f, Anf, n_exp, m_exp, f0, np0);
                nlist_term_f_lean<NE, ME, FORCE, ENERGY>(fb, gb_, gb, gb.q2 < rc2f, Anf, n_exp, m_exp, f1, SHIFT ? np1 : np0);
            } else {
                nlist_term_lean<NE, ME, FORCE, ENERGY>(pa, qa, rc2, An, n_exp, m_exp, acc0, np0);
                nlist_term_lean<NE, ME, FORCE, ENERGY>(pb, qb, rc2, An, n_exp, m_exp, acc1, SHIFT ? np1 : np0);
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
        auto gather = [&](const int *ip, double4 (&p)[CH]) {
#pragma unroll
            for (int u = 0; u < CH; ++u) {
                p[u] = load_record(recs + ip[32 * u]);
            }
        };
        auto compute = [&](const double4 (&p)[CH]) {
#pragma unroll
            for (int u = 0; u < CH; ++u) entry2(p[u], p[u]);
            flush();
        };
        // ---- whole iterations of CH batches: 2 CH independent chains per lane, no branches.  With kNlistPF the loop is
        //      unrolled by two so that two register sets alternate (no moves): the gathers of the next iteration are in
        //      flight while this one is in the pipe; past the last whole iteration the gather re-reads the last one. ----
        const int *ip = list + lane;
        if constexpr (!kListRuns && !kNlistPF) {
            static_assert(kNlistRW >= kNlistCH, "the words fetched a row ahead hold the first iteration's indices");
            int jc[CH], jn[CH];
#pragma unroll
            for (int u = 0; u < CH; ++u) jc[u] = int(rw[u]);
            for (int it = 0; it < nwhole; ++it) {
                const int *nx = ip + min(it + 1, nwhole - 1) * (32 * CH);   // indices of the next whole iteration, in flight
#pragma unroll
                for (int u = 0; u < CH; ++u) jn[u] = nx[32 * u];
                double4 pc[CH];
#pragma unroll
                for (int u = 0; u < CH; ++u) pc[u] = load_record(recs + jc[u]);
                compute(pc);
#pragma unroll
                for (int u = 0; u < CH; ++u) jc[u] = jn[u];
            }
        } else if constexpr (kNlistPF) {
            if (nwhole > 0) {
                double4 pA[CH], pB[CH];
                const int *last = ip + (nwhole - 1) * (32 * CH);
                gather(ip, pA);
                for (int it = 0; it < nwhole; it += 2) {
                    gather(ip + 32 * CH < last ? ip + 32 * CH : last, pB);
                    compute(pA);
                    if (it + 1 < nwhole) {
                        gather(ip + 64 * CH < last ? ip + 64 * CH : last, pA);
                        compute(pB);
                    }
                    ip += 64 * CH;
                }
            }
        } else {
            if constexpr (kNlistL1PF > 0) {
                // the first iterations' records (the list is padded, so reading a little past the whole iterations is harmless)
                const int ahead = min(kNlistL1PF * CH, nb32);
                for (int b = 0; b < ahead; ++b) prefetch_l1(recs + ip[32 * b]);
            }
            for (int it = 0; it < nwhole; ++it, ip += 32 * CH) {
                double4 pc[CH];
                if constexpr (kNlistL1PF > 0) {
                    if ((it + kNlistL1PF) * CH < nb32) {
#pragma unroll
                        for (int u = 0; u < CH; ++u)
                            if ((it + kNlistL1PF) * CH + u < nb32) prefetch_l1(recs + ip[32 * (kNlistL1PF * CH + u)]);
                    }
                }
                gather(ip, pc);
                compute(pc);
            }
        }
        // ---- the remaining 1 .. CH batches, one at a time; the last one carries the pair term in lane `lpair` ----
        for (int b = nwhole * CH; b < nb32; ++b) {
            const double4 p = load_record(recs + list[b * 32 + lane]);
            const bool pair_lane = b == nb32 - 1 && lane == lpair;
            const double4 qa = pair_lane ? pb : p, qb = pair_lane ? pa : p;
            entry2(qa, qb);
            flush();
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
                for (int b = 0; b < nb32; ++b) {
                    const bool pair_lane = b == nb32 - 1 && lane == lpair;
                    const int j = list[b * 32 + lane];
                    const int ja = pair_lane ? i1 : j, jb = pair_lane ? i0 : j;     // the record each atom meets
                    const double4 p = load_record(recs + j);
                    const double4 qa = pair_lane ? pb : p, qb = pair_lane ? pa : p;
                    const RecF &ga_ = reinterpret_cast<const RecF &>(qa), &gb_ = reinterpret_cast<const RecF &>(qb);
                    const bool in0 = ja < N && nlist_exact_in_range(a.xs, i0, ja, rc2);
                    const bool in1 = i1 < N && jb < N && nlist_exact_in_range(a.xs, i1, jb, rc2);
                    nlist_term_f_lean<NE, ME, FORCE, ENERGY>(fa, ga_, nlist_geom_f(fa, ga_), in0, Anf, n_exp, m_exp, f0, np0);
                    nlist_term_f_lean<NE, ME, FORCE, ENERGY>(fb, gb_, nlist_geom_f(fb, gb_), in1, Anf, n_exp, m_exp, f1, SHIFT ? np1 : np0);
                    // the flush points of the fast loops: after every whole iteration, after every remaining batch
                    if (b >= nwhole * CH || (b % CH) == CH - 1) flush();
                }
                flush();
            }
        }
        npairs += np0 + np1;
        if constexpr (!FORCE && SHIFT) {
            // per-atom neighbour counts over the 32 lanes (integers: exact), for the shifted density
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) {
                np0 += __shfl_xor_sync(0xffffffffu, np0, off);
                np1 += __shfl_xor_sync(0xffffffffu, np1, off);
            }
        }

        // ---- sums over the 32 lanes (fixed order), each total lands in its own lane, which stores it ----
        if constexpr (!FORCE) {
            double v[2] = {acc0[0], acc1[0]};
            transpose_sum<2>(v);
            const int h = lane >> 4, i = h ? i1 : i0;
            if ((lane & 15) == 0 && i < N) {
                // shifted cutoff: every in-range term loses r_c^-m
                const double rho = SHIFT ? a.c.am * fma(-double(h ? np1 : np0), a.shift_m, v[0]) : a.c.am * v[0];
                a.rho[i] = rho;
                const double root = rho > 0.0 ? sqrt(rho) : 0.0;           // reading Q9
                const double sp = rho > 0.0 ? a.c.Bm / root : 0.0;
                a.xs[i].w = sp;
                if constexpr (MIXED) a.xfr[i].s = float(sp);
                contrib += root;
            }
        } else {
            double v[8] = {acc0[0], acc0[1], acc0[2], acc0[3], acc1[0], acc1[1], acc1[2], acc1[3]};
            transpose_sum<8>(v);
            const int q = lane >> 2, h = q >> 2, c = q & 3, i = h ? i1 : i0;   // lane 4 q holds value q = (atom h, component c)
            if ((lane & 3) == 0 && i < N) {
                if (c < 3) a.force[3 * size_t(i) + c] = v[0];
                else contrib += v[0];
            }
        }
        nr = nr_next;
#pragma unroll
        for (int u = 0; u < RW; ++u) rw[u] = rw_next[u];
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
