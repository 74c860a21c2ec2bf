// scmd.cu -- host side of libscmd: context, workspace carving, kernel selection and launches.
// The C ABI is declared and documented in include/scmd.h.
#include "../../include/scmd.h"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <algorithm>
#include <functional>
#include <new>
#include <queue>
#include <vector>

#define SCMD_MAIN_TU 1   // this translation unit compiles the non-template kernels
#include "sc_dispatch.h"
#include "sc_device.cuh"
#include "sc_integrate.cuh"
#include "sc_small.cuh"
#include "sc_analysis.cuh"
#include "sc_allpairs_n3.cuh"

using namespace scmd;

namespace {

constexpr size_t kAlign = 256;
constexpr int kBlock = 256;          // O(N) kernels

struct Carver {
    unsigned char *base;
    size_t off = 0;
    explicit Carver(void *b) : base(static_cast<unsigned char *>(b)) {}
    template <class T>
    T *take(size_t count) {
        off = (off + kAlign - 1) / kAlign * kAlign;
        T *p = base ? reinterpret_cast<T *>(base + off) : nullptr;
        off += count * sizeof(T);
        return p;
    }
    size_t total() const { return (off + kAlign - 1) / kAlign * kAlign; }
};

inline int ceil_div(int64_t a, int64_t b) { return int((a + b - 1) / b); }

}  // namespace

struct sc_ctx {
    sc_params p{};
    int64_t N = 0;
    int row_begin = 0, row_end = 0;   // rows this context computes and integrates ([0, N) unless created as one rank of a row split)
    bool split = false;               // one rank of a row split over several GPUs (sc_step_rows)
    int32_t precision = 0;
    double skin = 0.0;
    cudaStream_t stream = nullptr;
    char err[512] = {0};
    int sm_count = 148;

    // device arrays (all inside the caller's workspace)
    double4 *xs = nullptr;        // [N] (x, y, z, s')
    unsigned long long *rdf_counts = nullptr;   // [kRdfMaxBins + 1] histogram; the last word is the reference-atom count
    int *rdf_refs = nullptr;      // [N] reference atoms of sc_rdf
    double *rdf_meta = nullptr;   // [4] centre
    double *msd_part = nullptr;   // [3 * kMsdMaxBlocks * kMsdPartStride] per-CTA partials of sc_msd
    double *msd_meta = nullptr;   // [kMsdMeta] centroids, rotation, totals
    double4 *n3_part = nullptr;   // Newton's-third-law sweeps: triangular reaction partials, row sums (else NULL)
    double4 *n3_self = nullptr;
    N3Tile *n3_tiles = nullptr;   // ... and their plan (plan_n3): tiles, first tile of each CTA's piece, slots per row block
    int *n3_piece_start = nullptr, *n3_blk_slots = nullptr;
    unsigned long long *n3_barrier = nullptr;      // grid barrier counter of n3_loop_kernel; the host tracks the value
    unsigned long long n3_barrier_count = 0;
    double *sprime = nullptr;     // [N] s' of the current step (one-launch step loop)
    unsigned long long *small_barrier = nullptr;   // its grid barrier counter; the host tracks the value
    unsigned long long small_barrier_count = 0;
    double4 *xs_b = nullptr;      // [N] second record buffer of the one-launch step loop (small all-pairs clusters)
    RecF *xfr = nullptr;          // [N + 1] split binary32 records (mixed list sweeps only)
    FPair *xf = nullptr;          // [(N + 512) / 2 + 1] packed split binary32 records (mixed all-pairs path only)
    double *vel = nullptr;        // [N*3]
    double *force = nullptr;      // [N*3]
    double *rho = nullptr;        // [N]
    double *part_a = nullptr;     // [max CTAs] per-CTA partials, sweep 1
    double *part_b = nullptr;     // [max CTAs] per-CTA partials, sweep 2
    double *part_ke = nullptr;    // [ceil(N/kBlock)]
    double *scal = nullptr;       // [kNumScalars]
    double *stage_a = nullptr;    // [N*3] host-path staging
    double *stage_b = nullptr;    // [N*3]

    // cutoff path (r_cut > 0); all null otherwise
    bool cutoff = false;
    double r_list = 0.0;
    int kmax = 0, kmax_cap = 0, max_dim = 1, coop_grid = 0, small_ctas = 0;
    bool list_checked = false;    // rebuild_kernel already launched for the current positions
    bool pairs_zeroed = false;    // ... and it zeroed the in-range pair counter for the density sweep that follows
    double4 *xs_alt = nullptr, *xs_ref = nullptr;
    double *vel_alt = nullptr, *blockpart = nullptr;
    int *perm = nullptr, *perm_alt = nullptr, *cell_of = nullptr, *slot_of = nullptr, *cell_sorted = nullptr;
    int *cell_count = nullptr, *cell_start = nullptr, *order_tmp = nullptr, *order = nullptr;
    int *nlist = nullptr, *ncount = nullptr, *scanpart = nullptr;
    CellGrid *grid = nullptr;
    unsigned long long *counters = nullptr;

    PairConsts consts{};
    bool have_pos = false, have_vel = false;
    bool density_valid = false, forces_valid = false, energy_valid = false;
    bool lambda_pending = false;
    int64_t launches = 0;
    uint64_t langevin_step = 0;   // generator step of the next Langevin update (SC_OPT_LANGEVIN_STEP)

    struct OccEntry { const void *fn; int warps; int per_sm; };
    std::vector<OccEntry> occ_cache;

    // options (0 = default)
    int opt_it = 0, opt_tpr = 0, opt_warps = 0, opt_persistent = 0, opt_energy_every = 0, opt_kmax = 0, opt_fine = 0, opt_apc = 0, opt_n3 = 0, opt_shift = 0;
    int emb_pending = 0;          // sweep 1 left this many per-CTA sums of sqrt(rho) in part_a, not yet totalled into U_emb
    int n3_seg = 0;               // Newton's-third-law sweeps: CTAs (= pieces) of the plan on the device; 0 = no plan yet
    int opt_n3_pieces = 0;
    int n3_warps = 12;            // ... and their warps per CTA (12, or 6 with two CTAs per SM)
    int n3_fuse = 0;              // do_step -> run_sweep_n3: what the force finalize kernel integrates (N3FinalArgs::fuse)
    double n3_hk = 0.0, n3_dt = 0.0;

    // profiling
    bool profile = false;
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
    double ms_density = 0, ms_force = 0, ms_other = 0;
};

namespace {

sc_status fail(sc_ctx *c, sc_status st, const char *fmt, const char *detail = "") {
    if (c) snprintf(c->err, sizeof(c->err), fmt, detail);
    return st;
}

#define SC_CUDA_CHECK(ctx, call)                                                     \
    do {                                                                             \
        cudaError_t e_ = (call);                                                     \
        if (e_ != cudaSuccess) return fail((ctx), SC_ERR_CUDA, #call ": %s", cudaGetErrorString(e_)); \
    } while (0)

bool params_ok(const sc_params *p) {
    return p && p->n > p->m && p->m > 0 && p->n <= 64 && p->eps > 0.0 && p->a > 0.0 && p->mass > 0.0 &&
           std::isfinite(p->eps) && std::isfinite(p->a) && std::isfinite(p->c) && std::isfinite(p->mass) &&
           std::isfinite(p->r_cut);
}

bool create_options_ok(const sc_create_options *o) {
    if (!o) return true;
    for (int r : o->reserved)
        if (r != 0) return false;
    return o->neighbour_capacity >= 0 && (o->newton3_storage == 0 || o->newton3_storage == 2) && o->row_begin >= 0 &&
           o->row_end >= o->row_begin;
}
bool row_split(const sc_create_options *o) { return o && o->row_end > o->row_begin; }

constexpr int kMaxCoopBlocks = 4096;

inline int round_up(int64_t v, int64_t q) { return int((v + q - 1) / q * q); }

// default neighbour-row capacity: 1.3 x the fcc number density 4 / a^3 inside the list sphere
int default_kmax(const sc_params *p, int64_t N, double skin) {
    const double rl = p->r_cut + skin;
    const double est = 1.3 * (4.0 / (p->a * p->a * p->a)) * (4.0 / 3.0) * 3.14159265358979323846 * rl * rl * rl;
    int64_t k = int64_t(est) + 1;
    if (k > N - 1) k = N - 1;
    if (k < 1) k = 1;
    return round_up(k, 32);
}
// cell budget: fine cells of edge r_list / 4 hold ~2 atoms at metallic densities and a sphere fills half
// of its bounding box, so ~N cells are needed; 4 N leaves room for dilute clusters
int cutoff_max_dim(int64_t N) {
    const int64_t cap = 4 * N + 4096;
    int d = 1;
    while (int64_t(d + 1) * (d + 1) * (d + 1) <= cap) ++d;
    return d;
}

// Newton's-third-law all-pairs sweeps (sc_allpairs_n3.cuh): sizes for which their partial sums are carved
constexpr int64_t kN3MinAtoms = 2048, kN3MaxAtoms = 262144;   // workspace carved in this range (4.3 GB at the top)
constexpr int64_t kN3DefaultMinAtoms = 2961, kN3DefaultMinAtomsMixed = 2961;   // measured crossovers
constexpr int kN3RowsPerThread = 4;     // 2 rows per lane (twice the chunks, half as long) measured in the step loop for small
                                        // clusters, where the triangle has fewer chunks than the chip has warps: N = 2057 23.4
                                        // against 24.8, N = 2304 23.3 / 24.3, N = 3072 33.2 / 30.3, N = 4096 48.9 / 38.9 us per step
constexpr int kN3PairRows = 64 * kN3RowsPerThread;             // rows of a pair block (two row sets per CTA: sc_allpairs_n3.cuh)
constexpr int kN3MaxSegments = 25;                             // j segments (tiles) of the longest row block
constexpr int kN3MaxPieces = 4096;                             // CTAs of a balanced plan (16 per SM on 256 SMs)
inline size_t n3_tile_capacity(int64_t N) {                    // the round-1 grid has up to 25 tiles per row block
    return size_t(ceil_div(N, int64_t(32 * kN3RowsPerThread))) * kN3MaxSegments + kN3MaxPieces;
}

// one place that lays the workspace out; base == nullptr only measures
size_t carve(sc_ctx *c, void *base, int64_t N, const sc_params *prm, int32_t precision, double skin,
             const sc_create_options *opt) {
    Carver w(base);
    const size_t n = size_t(N);
    double4 *xs = w.take<double4>(n + kTileAtoms);
    double *vel = w.take<double>(3 * n);
    double *force = w.take<double>(3 * n);
    double *rho = w.take<double>(n);
    double *pa = w.take<double>(n + 1);
    double *pb = w.take<double>(n + 1);
    double *pk = w.take<double>(size_t(ceil_div(N, kBlock)) + 1 + 1024);   // also the per-CTA partials of the one-launch loop
    double *scal = w.take<double>(kNumScalars);
    double *sa = w.take<double>(3 * n);
    double *sb = w.take<double>(3 * n);
    unsigned long long *rc = w.take<unsigned long long>(kRdfMaxBins + 2);
    int *rr = w.take<int>(n);
    double *rm = w.take<double>(4);
    double *mp = w.take<double>(size_t(3) * kMsdMaxBlocks * kMsdPartStride);
    double *mm = w.take<double>(kMsdMeta);
    if (c && base) {
        c->xs = xs; c->vel = vel; c->force = force; c->rho = rho; c->part_a = pa; c->part_b = pb;
        c->part_ke = pk; c->scal = scal; c->stage_a = sa; c->stage_b = sb;
        c->rdf_counts = rc; c->rdf_refs = rr; c->rdf_meta = rm; c->msd_part = mp; c->msd_meta = mm;
    }
    if (!(prm->r_cut > 0.0) && N <= kSmallMaxAtoms && !row_split(opt)) {
        double4 *xb = w.take<double4>(n + 8);                  // staged layout: whole blocks of 8 records (sc_small.cuh)
        double *spr = w.take<double>(n);
        unsigned long long *bar = w.take<unsigned long long>(2);
        if (c && base) { c->xs_b = xb; c->sprime = spr; c->small_barrier = bar; }
    }
    if (!(prm->r_cut > 0.0) && N >= kN3MinAtoms && N <= kN3MaxAtoms && !(opt && opt->newton3_storage == 2) && !row_split(opt)) {
        double4 *np = w.take<double4>(n3_part_records(int(N), kN3PairRows));
        double4 *ns = w.take<double4>((n + 32) * kN3MaxSegments);
        RecF *xr = precision == SC_PREC_MIXED ? w.take<RecF>(n + 1) : nullptr;    // split records of the mixed variant
        N3Tile *tl = w.take<N3Tile>(n3_tile_capacity(N));
        int *ps = w.take<int>(n3_tile_capacity(N) + 1);
        int *bs = w.take<int>(size_t(ceil_div(N, int64_t(32 * kN3RowsPerThread))));
        unsigned long long *nbar = w.take<unsigned long long>(2);
        if (c && base) {
            c->n3_part = np; c->n3_self = ns; c->n3_tiles = tl; c->n3_piece_start = ps; c->n3_blk_slots = bs; c->n3_barrier = nbar;
            if (xr) c->xfr = xr;
        }
    }
    if (precision == SC_PREC_MIXED && !(prm->r_cut > 0.0)) {
        FPair *xf = w.take<FPair>((n + kTileAtoms) / 2 + 1);
        if (c && base) c->xf = xf;
    }
    if (prm->r_cut > 0.0) {
        const int kmax = opt && opt->neighbour_capacity > 0
                             ? round_up(std::min<int64_t>(opt->neighbour_capacity, std::max<int64_t>(N - 1, 1)), 32)
                             : default_kmax(prm, N, skin);
        const int md = cutoff_max_dim(N);
        const size_t ncell = size_t(md) * md * md + 2;
        double4 *xa = w.take<double4>(n + kTileAtoms);
        RecF *xfr = precision == SC_PREC_MIXED ? w.take<RecF>(n + 1) : nullptr;
        double4 *xr = w.take<double4>(n);
        double *va = w.take<double>(3 * n);
        double *bp = w.take<double>(9 * size_t(kMaxCoopBlocks));
        int *perm = w.take<int>(n), *perm_alt = w.take<int>(n), *cell_of = w.take<int>(n), *slot_of = w.take<int>(n);
        int *cell_sorted = w.take<int>(n), *order_tmp = w.take<int>(n), *order = w.take<int>(n), *ncount = w.take<int>(n);
        int *cell_count = w.take<int>(ncell), *cell_start = w.take<int>(ncell);
        int *nlist = w.take<int>(size_t(kmax) * (n + 1));      // ceil(N / 2) pair rows of 2 kmax entries
        int *scanpart = w.take<int>(size_t(kMaxCoopBlocks) + 1);
        CellGrid *grid = w.take<CellGrid>(1);
        unsigned long long *counters = w.take<unsigned long long>(kNumCounters);
        if (c && base) {
            c->xs_alt = xa; c->xfr = xfr; c->xs_ref = xr; c->vel_alt = va; c->blockpart = bp; c->perm = perm; c->perm_alt = perm_alt;
            c->cell_of = cell_of; c->slot_of = slot_of; c->cell_sorted = cell_sorted; c->order_tmp = order_tmp;
            c->order = order; c->ncount = ncount; c->cell_count = cell_count; c->cell_start = cell_start;
            c->nlist = nlist; c->scanpart = scanpart; c->grid = grid; c->counters = counters;
            c->kmax = c->kmax_cap = kmax; c->max_dim = md;
        }
    }
    return w.total();
}

double ipow_host(double u, int k) {
    double r = 1.0;
    for (int t = 0; t < k; ++t) r *= u;
    return r;
}

// ---------------------------------------------------------------------------------------------
// all-pairs kernel selection
// ---------------------------------------------------------------------------------------------
struct TileChoice { int it, tpr, warps; };

const void *allpairs_fn(const sc_ctx *c, int it, int tpr, bool force, bool energy) {
    const bool fast = (c->p.n == 9 && c->p.m == 6), mixed = c->precision == SC_PREC_MIXED;
    if (mixed) return fast ? allpairs32_fn_96(it, tpr, force, energy) : allpairs32_fn_generic(it, tpr, force, energy);
    return fast ? allpairs64_fn_96(it, tpr, force, energy) : allpairs64_fn_generic(it, tpr, force, energy);
}

// resident CTAs per SM of one instantiation at (warps + 1) * 32 threads; cached per context
int allpairs_residency(sc_ctx *c, const void *fn, int it, int tpr, int warps) {
    const size_t smem = allpairs_smem_bytes(it, tpr, warps);
    for (const auto &e : c->occ_cache)
        if (e.fn == fn && e.warps == warps) return e.per_sm;
    int per_sm = 1;
    if (cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem)) != cudaSuccess ||
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, (warps + 1) * 32, smem) != cudaSuccess || per_sm < 1)
        per_sm = 1;
    c->occ_cache.push_back({fn, warps, per_sm});
    return per_sm;
}

// Tile shape for one sweep.  Rows per CTA = 32 / tpr * it.
//  * N >= 7104 (measured sweep over it x tpr x warps at N = 8000 ... 262144): 4 consumer warps per
//    CTA and the largest row block among 64 (4 rows per thread, 2 lanes per row), 32 (4, 4), 16 (2, 4) that
//    still gives >= 6 CTAs per SM; 4 rows per thread put 16 independent pair chains in flight per thread, which
//    the FP64 pipe needs more than it needs resident warps (3-8 % over 2 rows per thread and 8 warps);
//  * smaller N: CTAs run in waves of sm_count * residency, and a partly filled last wave idles the chip, so among
//    the shapes with 2 rows per thread take the one whose wave efficiency x / ceil(x) is best, preferring more
//    rows per CTA when it is a tie (x < 1: efficiency = x, i.e. the shape with the most CTAs, down to one row
//    per CTA), discounted for the lanes that split j inside a warp.
TileChoice choose_tile(sc_ctx *c, bool force, bool energy) {
    const int64_t N = c->row_end - c->row_begin;       // rows to cover (the j range is always all atoms)
    TileChoice best{2, 1, 8};
    int warps_pref = 0;
    if (c->opt_it && c->opt_tpr) {
        best.it = c->opt_it; best.tpr = c->opt_tpr;
    } else if (!c->opt_it && !c->opt_tpr && N >= 3 * 16 * int64_t(c->sm_count) &&
               (c->precision != SC_PREC_MIXED || N >= 6 * 64 * int64_t(c->sm_count))) {
        static const int shapes[3][2] = {{4, 2}, {4, 4}, {2, 4}};
        best.it = 2; best.tpr = 4;
        for (const auto &sh : shapes) {
            if (!allpairs_fn(c, sh[0], sh[1], force, energy)) continue;
            if (ceil_div(N, allpairs_rows_per_cta(sh[0], sh[1])) >= 6 * c->sm_count) { best.it = sh[0]; best.tpr = sh[1]; break; }
        }
        warps_pref = 4;
    } else {
        double best_eff = -1.0;
        const int its[2] = {2, 1};
        for (int it : its) {
            if (c->opt_it && it != c->opt_it) continue;
            for (int tpr = 1; tpr <= 32; tpr *= 2) {
                if (c->opt_tpr && tpr != c->opt_tpr) continue;
                if (it == 1 && tpr != 32 && !c->opt_it) continue;       // 1 row per thread only as the smallest shape
                const void *fn = allpairs_fn(c, it, tpr, force, energy);
                if (!fn) continue;
                const int rpc = allpairs_rows_per_cta(it, tpr);
                const double x = double(ceil_div(N, rpc)) / (double(c->sm_count) * allpairs_residency(c, fn, it, tpr, 8));
                // lanes that split j inside a warp cost shared-memory bandwidth and epilogue shuffles (measured)
                static const double lanes64[6] = {1.0, 1.0, 0.97, 0.90, 0.75, 0.6}, lanes32[6] = {1.0, 0.92, 0.75, 0.5, 0.35, 0.25};
                const int lg = tpr == 1 ? 0 : tpr == 2 ? 1 : tpr == 4 ? 2 : tpr == 8 ? 3 : tpr == 16 ? 4 : 5;
                const double eff = x / std::ceil(x) * (c->precision == SC_PREC_MIXED ? lanes32[lg] : lanes64[lg]);
                if (eff > best_eff + 0.02) { best_eff = eff; best.it = it; best.tpr = tpr; }
            }
        }
        if (c->opt_it) best.it = c->opt_it;
        if (c->opt_tpr) best.tpr = c->opt_tpr;
    }
    int warps = warps_pref ? warps_pref : 8;
    while (warps > 1 && c->N / (int64_t(warps) * best.tpr) < 8) warps /= 2;   // >= ~8 pairs per lane and row
    if (c->opt_warps) warps = c->opt_warps;
    best.warps = warps;
    return best;
}

// ---------------------------------------------------------------------------------------------
// cutoff path: rebuild + list-driven sweeps
// ---------------------------------------------------------------------------------------------
sc_status ensure_list(sc_ctx *c) {
    if (!c->cutoff || c->list_checked) return SC_OK;
    RebuildArgs a{};
    a.xs = c->xs; a.xs_alt = c->xs_alt; a.xs_ref = c->xs_ref; a.xfr = c->xfr; a.vel = c->vel; a.vel_alt = c->vel_alt;
    a.perm = c->perm; a.perm_alt = c->perm_alt; a.cell_of = c->cell_of; a.slot_of = c->slot_of;
    a.cell_sorted = c->cell_sorted; a.cell_count = c->cell_count; a.cell_start = c->cell_start;
    a.order_tmp = c->order_tmp; a.order = c->order; a.nlist = c->nlist; a.ncount = c->ncount;
    a.blockpart = c->blockpart; a.scanpart = c->scanpart; a.grid = c->grid; a.scal = c->scal; a.counters = c->counters;
    a.n_atoms = int(c->N); a.kmax = c->kmax; a.max_dim = c->max_dim;
    a.fine_max = c->opt_fine ? c->opt_fine : kFineMax;
    a.have_vel = c->have_vel ? 1 : 0;
    a.zero_pairs = c->density_valid ? 0 : 1;            // the density sweep that follows counts from zero
    a.r_list = c->r_list; a.half_skin2 = 0.25 * c->skin * c->skin;
    void *params[] = {&a};
    cudaError_t e = cudaLaunchCooperativeKernel(reinterpret_cast<void *>(rebuild_kernel), dim3(c->coop_grid), dim3(256),
                                                params, 0, c->stream);
    if (e != cudaSuccess) return fail(c, SC_ERR_CUDA, "rebuild_kernel launch: %s", cudaGetErrorString(e));
    c->launches += 1;
    c->list_checked = true;
    c->pairs_zeroed = a.zero_pairs != 0;
    return SC_OK;
}

// list sweeps: warps per CTA and consecutive atom pairs per CTA.  The warps of a CTA work on adjacent
// pairs at the same time, so the records they gather are the same L1 lines.
int choose_nlist_warps(const sc_ctx *c) { return c->opt_warps ? c->opt_warps : 4; }
int choose_pairs_per_cta(const sc_ctx *c, int warps) {
    int64_t ppc = c->opt_apc ? (c->opt_apc + 1) / 2 : 2 * warps;
    ppc = ppc / warps * warps;
    return int(ppc < warps ? warps : ppc);
}
// grid of the list sweeps: CTA c takes the row blocks c, c + grid, ...  Measured at N = 65536: one
// resident wave (6 CTAs per SM) and one CTA per block perform alike (84.7 + 105.5 against 82.5 + 104.2 us); the cap
// only keeps the per-CTA partial sums few at N = 2^20.
int choose_nlist_grid(const sc_ctx *c, int ppc) {
    const int blocks = ceil_div((c->N + 1) / 2, ppc);
    return std::min(blocks, c->sm_count * 32);
}

sc_status run_sweep_cutoff(sc_ctx *c, bool force, bool energy) {
    sc_status st = ensure_list(c);
    if (st != SC_OK) return st;
    NlistArgs a{};
    a.xs = c->xs; a.xfr = c->xfr; a.nlist = c->nlist; a.ncount = c->ncount; a.n_atoms = int(c->N); a.kmax = c->kmax;
    const int warps = choose_nlist_warps(c);
    a.pairs_per_cta = choose_pairs_per_cta(c, warps);
    a.idx_cap = 2 * c->kmax + 64;
    a.rho = c->rho; a.force = c->force; a.partial = force ? c->part_b : c->part_a;
    a.pairs_in_cut = c->counters + kCntPairsInCut;
    a.rc2 = c->p.r_cut * c->p.r_cut;
    a.shift_m = c->opt_shift ? ipow_host(1.0 / c->p.r_cut, c->p.m) : 0.0;
    a.c = c->consts;
    if (!force) {
        if (!c->pairs_zeroed)
            SC_CUDA_CHECK(c, cudaMemsetAsync(c->counters + kCntPairsInCut, 0, sizeof(unsigned long long), c->stream));
        c->pairs_zeroed = false;
    }
    const bool fast = (c->p.n == 9 && c->p.m == 6), mixed = c->precision == SC_PREC_MIXED;
    const int grid = choose_nlist_grid(c, a.pairs_per_cta);
    cudaError_t e = fast ? launch_nlist_96(grid, warps * 32, a, force, energy, mixed, c->stream)
                         : launch_nlist_generic(grid, warps * 32, a, force, energy, mixed, c->stream);
    if (e != cudaSuccess) return fail(c, SC_ERR_CUDA, "list sweep launch: %s", cudaGetErrorString(e));
    c->launches += 1;
    if (!force || energy) {
        if (!force) {
            c->emb_pending = grid;                                // totalled when an energy is asked for (ensure_forces)
        } else {
            if (c->opt_shift)
                reduce_partials_shift_kernel<<<1, 1024, 0, c->stream>>>(a.partial, grid, c->scal, kSlotEPair, c->consts.En,
                                                                       c->counters + kCntPairsInCut,
                                                                       ipow_host(1.0 / c->p.r_cut, c->p.n));
            else
                reduce_partials_kernel<<<1, 1024, 0, c->stream>>>(a.partial, grid, c->scal, kSlotEPair, c->consts.En);
            SC_CUDA_CHECK(c, cudaGetLastError());
            c->launches += 1;
        }
    }
    return SC_OK;
}

// device flags raised by the cutoff path; call after a stream synchronisation point
sc_status check_flags(sc_ctx *c) {
    if (!c->cutoff) return SC_OK;
    unsigned long long cnt[kNumCounters];
    SC_CUDA_CHECK(c, cudaMemcpyAsync(cnt, c->counters, sizeof(cnt), cudaMemcpyDeviceToHost, c->stream));
    SC_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    if (cnt[kCntOverflow])
        return fail(c, SC_ERR_CAPACITY, "a neighbour row overflowed its capacity; results since then are invalid%s");
    return SC_OK;
}

// GRID PLAN ONLY (SC_OPT_NEWTON3_PIECES = -1; the default is the balanced plan of plan_n3 below).
// Segment length of the Newton's-third-law sweeps, in chunks of 32 atoms.  Their CTAs (row block x j segment; one CTA
// per SM at 168 registers x 384 threads) are handed to the SMs in launch order as SMs fall free, so the sweep lasts as
// long as the busiest SM of that greedy schedule: with a few hundred CTAs on 148 SMs a badly filled last wave costs
// 10 % (measured at N = 8000 ... 24576, where the best of 8 / 12 / 16 / 24 segments changes with N in no simple way).
// The schedule is simulated for each candidate -- a CTA costs one unit of prologue / epilogue plus one per round of its
// 12 warps over the segment's chunks (mixed: chunks of 64, and a quarter unit of fixed cost: calibrated) -- and the
// shortest makespan wins.  Against measurement the simulation picked the fastest candidate at 6 (FP64) and 5 (mixed)
// of 8 sizes between 7000 and 32768 and was within 1 - 6 % at the others; above 49152 the choice is flat within 1 %.
// Returns the segment length; *warps_out = warps per CTA: 12.  TWO CTAs of 6 warps per SM (same registers, tiles half as
// large, twice the slots: by this simulation the cure for N = 8000, where 252 tiles fill 296 slot-rounds to 80 %) were
// measured in round 2 (both resident) and are SLOWER (200-step calls: N = 6144 120 against 102, N = 8000 217 against 140,
// N = 16384 479 against 401 us per step: a tile lasts as long as its slowest warp, and with 3 chunks per warp one diagonal chunk decides):
// SC_OPT_WARPS_PER_CTA <= 6 still selects them, the default never does.
int choose_n3_segment(const sc_ctx *c, int *warps_out) {
    const int N = int(c->N), nch = ceil_div(N, 32), nb = ceil_div(N, 32 * kN3RowsPerThread);
    const int unit = c->precision == SC_PREC_MIXED ? 2 : 1;
    const double fixed = c->precision == SC_PREC_MIXED ? 0.25 : 1.0;
    int best_seg = 0, best_w = kN3Warps;
    double best_t = 0.0;
    for (int nw : {kN3Warps, kN3Warps / 2}) {
        if (nw != ((c->opt_warps && c->opt_warps <= 6) ? 6 : 12)) continue;    // SC_OPT_WARPS_PER_CTA <= 6 forces 6
        // candidates: every segment length that is a whole number of rounds of the CTA's warps and gives <= 25 segments
        // (round 1 tried only 8 / 12 / 16 / 20 / 24 segments; for a mid-size cluster ONE tile per SM -- 3 or 4 long
        // segments -- beats two short rounds: bench steps N = 6144 0.127 -> 0.108 ms, 8000 0.165 -> 0.161, 16384 0.425 -> 0.408,
        // mixed 8000 0.140 -> 0.133).  Beyond 16384 atoms (mixed: 8192) the fine set measured 2 - 3 % WORSE than the coarse one
        // (the cost model is not that good), and above 49152 the choice is flat within 1 %.
        std::vector<int> cands;
        if (N > (c->precision == SC_PREC_MIXED ? 8192 : 16384)) {
            for (int want : {8, 12, 16, 20, 24}) cands.push_back(round_up(ceil_div(nch, want), nw * unit));
        } else {
            for (int seg = nw * unit; seg < nch + nw * unit; seg += nw * unit) cands.push_back(seg);
        }
        int last_seg = 0;
        for (int seg : cands) {
            const int nseg = ceil_div(nch, seg);
            if (nseg > kN3MaxSegments || seg == last_seg) continue;
            last_seg = seg;
            std::priority_queue<double, std::vector<double>, std::greater<double>> sm;
            for (int k = 0; k < c->sm_count * (kN3Warps / nw); ++k) sm.push(0.0);
            double makespan = 0.0;
            for (int y = 0; y < nseg; ++y)
                for (int b = 0; b < nb; ++b) {
                    const int c_begin = b * kN3RowsPerThread + y * seg;
                    if (c_begin >= nch) continue;
                    const int chunks = ceil_div(std::min(nch, c_begin + seg) - c_begin, unit);
                    // a CTA of nw warps shares its SM's pipes with 12 / nw - 1 others: per-warp progress is the same
                    const double t = sm.top() + fixed + double(ceil_div(chunks, nw));
                    sm.pop();
                    sm.push(t);
                    makespan = std::max(makespan, t);
                }
            if (!best_seg || makespan < best_t - 1e-9) { best_seg = seg; best_t = makespan; best_w = nw; }
        }
    }
    *warps_out = best_w;
    return best_seg;
}

// The plan of the Newton's-third-law sweeps: which CTA works through which tiles (sc_allpairs_n3.cuh, N3Tile).
//
// Balanced plan (the default).  The triangle, row block after row block, is cut into P = SMs x k pieces of equal COST,
// one CTA each; k = 1 (one wave of resident CTAs: nothing is left to the order in which SMs fall free; measured against
// k = 2 / 4 / 8 per SM, SC_OPT_NEWTON3_PIECES: N = 8000 103.7 / 110.1 us per step, N = 65536 5158 / 5157 / 5161 / 5180).
// Cost of a tile of L chunks of a PAIR block (2 x 128 rows, sc_allpairs_n3.cuh): ceil(L / 2) -- a chunk occupies two warps,
// one per row set; the six warp pairs take the chunks round-robin and land three to an SM sub-partition, so the tile lasts
// as long as the ceil(L / 2) chunk rotations of its busiest sub-partition (before the pair blocks: ceil(L / 4) for
// 12 warps on 128 rows) -- plus a fixed 0.15 for the tile's row loads and its reduction (two CTA barriers).  The smallest cost bound T for which the greedy cut (fill a piece up to T, never with a sliver
// shorter than 4 chunks unless it ends the row block) needs <= P pieces is found by bisection.  N = 8000: 7938 chunks
// on 148 SMs = 13.4 per sub-partition, the plan gives every CTA <= 14; the round-1 grid gave the longest 18 (6 rounds x
// 3 warps) and the sweep lasted 78 us where 14 / 18 of that is 61 -- measured 61.2 (300-step calls, us per step, grid
// plan -> balanced: N = 6144 73.7 -> 71.8, N = 8000 123.3 -> 103.7, mixed 99.0 -> 86.1, N = 16384 360.5 -> 346.9,
// N = 65536 5251 -> 5158, mixed 3981 -> 3909).
//
// Grid plan (SC_OPT_NEWTON3_PIECES = -1; rounds 1 - 2a, kept for comparison): one tile per CTA, row block x j segment
// with ONE segment length for all row blocks (choose_n3_segment), CTAs in launch order.
struct N3Plan {
    std::vector<N3Tile> tiles;
    std::vector<int> piece_start, blk_slots;
};

// greedy cut for the cost bound T; false if it needs more than max_pieces pieces or a row block more than 25 tiles
bool n3_cut(int nb, int nch, int cpb, double T, double fixed, int max_pieces, N3Plan *out) {
    out->tiles.clear(); out->piece_start.assign(1, 0); out->blk_slots.assign(size_t(nb), 0);
    double cur = 0.0;
    auto close = [&]() {
        if (int(out->tiles.size()) > out->piece_start.back()) out->piece_start.push_back(int(out->tiles.size()));
        cur = 0.0;
    };
    for (int b = 0; b < nb; ++b) {
        int cpos = b * cpb, slot = 0;
        while (cpos < nch) {
            const int rest = nch - cpos;
            const double room = T - cur - fixed;
            int fit = room >= 1.0 ? 2 * int(room + 1e-9) : 0;
            if (fit < rest && fit < 4) fit = 0;
            if (fit <= 0) {
                if (cur == 0.0) return false;                  // T below one tile's cost
                close();
                continue;
            }
            const int len = std::min(fit, rest);
            if (slot >= kN3MaxSegments) return false;
            out->tiles.push_back(N3Tile{b, cpos, cpos + len, slot++});
            cur += fixed + double(ceil_div(len, 2));
            cpos += len;
        }
        out->blk_slots[size_t(b)] = slot;
    }
    close();
    return int(out->piece_start.size()) - 1 <= max_pieces;
}

int choose_n3_segment(const sc_ctx *c, int *warps_out);

sc_status plan_n3(sc_ctx *c) {
    const int N = int(c->N), rb = kN3PairRows, nb = ceil_div(N, rb);   // pair blocks
    const bool mixed = c->precision == SC_PREC_MIXED;
    const int chunk = mixed ? 64 : 32, nch = ceil_div(N, chunk), cpb = rb / chunk;
    N3Plan plan;
    c->n3_warps = (c->opt_warps && c->opt_warps <= 6) ? 6 : kN3Warps;
    if (c->opt_n3_pieces < 0) {
        int warps = kN3Warps;
        const int seg32 = choose_n3_segment(c, &warps), seg = seg32 * 32 / chunk, nseg = ceil_div(ceil_div(N, 32), seg32);
        c->n3_warps = warps;
        plan.piece_start.assign(1, 0); plan.blk_slots.assign(size_t(nb), 0);
        for (int y = 0; y < nseg; ++y)
            for (int b = 0; b < nb; ++b) {
                const int c_begin = b * cpb + y * seg;
                if (c_begin >= nch) continue;
                plan.tiles.push_back(N3Tile{b, c_begin, std::min(nch, c_begin + seg), y});
                plan.piece_start.push_back(int(plan.tiles.size()));
                plan.blk_slots[size_t(b)] = y + 1;
            }
    } else {
        const int per_sm = c->opt_n3_pieces ? c->opt_n3_pieces : 1;
        const int P = std::min(std::min(kN3MaxPieces, N / 2), c->sm_count * (kN3Warps / c->n3_warps) * per_sm);   // part_b holds N + 1
        const double fixed = 0.15;
        double total = 0.0;
        for (int b = 0; b < nb; ++b) total += fixed + double(ceil_div(nch - b * cpb, 2));
        double lo = 1.0, hi = total + 2.0;                          // hi: everything in one piece, always feasible
        N3Plan trial;
        for (int it = 0; it < 48; ++it) {
            const double mid = 0.5 * (lo + hi);
            if (n3_cut(nb, nch, cpb, mid, fixed, P, &trial)) hi = mid; else lo = mid;
        }
        if (!n3_cut(nb, nch, cpb, hi, fixed, P, &plan))
            return fail(c, SC_ERR_INVALID, "Newton's-third-law sweeps: no plan for this size%s");
    }
    const int pieces = int(plan.piece_start.size()) - 1;
    if (plan.tiles.size() > n3_tile_capacity(c->N) || pieces < 1)
        return fail(c, SC_ERR_INVALID, "Newton's-third-law sweeps: plan exceeds the workspace carved for it%s");
    SC_CUDA_CHECK(c, cudaMemcpyAsync(c->n3_tiles, plan.tiles.data(), plan.tiles.size() * sizeof(N3Tile), cudaMemcpyHostToDevice, c->stream));
    SC_CUDA_CHECK(c, cudaMemcpyAsync(c->n3_piece_start, plan.piece_start.data(), plan.piece_start.size() * sizeof(int), cudaMemcpyHostToDevice, c->stream));
    SC_CUDA_CHECK(c, cudaMemcpyAsync(c->n3_blk_slots, plan.blk_slots.data(), plan.blk_slots.size() * sizeof(int), cudaMemcpyHostToDevice, c->stream));
    SC_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));           // the vectors die with this call
    c->n3_seg = pieces;
    return SC_OK;
}

// all pairs, every unordered pair once (sc_allpairs_n3.cuh): sweep + finalize + scalar reduction
sc_status run_sweep_n3(sc_ctx *c, bool force, bool energy) {
    const bool fast = (c->p.n == 9 && c->p.m == 6);
    const int it = kN3RowsPerThread, rb = kN3PairRows, N = int(c->N);   // measured: 2 rows per thread lose 10 % at N = 65536
    const void *fn = allpairs_n3_fn(it, fast, force, energy);
    const int nb = ceil_div(N, rb);
    const bool mixed = c->precision == SC_PREC_MIXED;
    if (mixed) fn = allpairs_n3p_fn(it, fast, force, energy);
    if (!fn) return fail(c, SC_ERR_INVALID, "Newton's-third-law sweep: no kernel for this shape%s");
    N3Args a{};
    a.xs = c->xs; a.n_atoms = N; a.n_pad = round_up(N, 32);
    a.part = c->n3_part; a.part_rho = reinterpret_cast<double *>(c->n3_part); a.self = c->n3_self;
    a.partial = c->part_b; a.c = c->consts;
    N3FArgs af{};
    af.xfr = c->xfr; af.n_atoms = N; af.n_pad = a.n_pad; af.part = a.part; af.part_rho = a.part_rho; af.self = a.self;
    if (!c->n3_seg) {
        sc_status st = plan_n3(c);
        if (st != SC_OK) return st;
    }
    const int pieces = c->n3_seg;
    a.tiles = c->n3_tiles; a.piece_start = c->n3_piece_start;
    af.partial = a.partial; af.c = a.c; af.tiles = a.tiles; af.piece_start = a.piece_start;
    void *params[1] = {mixed ? static_cast<void *>(&af) : static_cast<void *>(&a)};
    if (c->n3_warps < kN3Warps)       // two CTAs of 6 warps per SM need 2 x 37 KB of shared memory
        cudaFuncSetAttribute(fn, cudaFuncAttributePreferredSharedMemoryCarveout, int(cudaSharedmemCarveoutMaxShared));
    cudaError_t e = cudaLaunchKernel(fn, dim3(pieces), dim3(c->n3_warps * 32), params, 0, c->stream);
    if (e != cudaSuccess) return fail(c, SC_ERR_CUDA, "Newton's-third-law sweep launch: %s", cudaGetErrorString(e));
    N3FinalArgs f{};
    f.xs = c->xs; f.xfr = mixed ? c->xfr : nullptr; f.xf = mixed ? c->xf : nullptr; f.part = c->n3_part; f.part_rho = a.part_rho; f.self = c->n3_self; f.rho = c->rho; f.force = c->force;
    f.partial = c->part_a; f.n_atoms = N; f.n_pad = a.n_pad; f.rb = rb; f.blk_slots = c->n3_blk_slots; f.c = c->consts;
    f.fuse = force ? c->n3_fuse : 0; f.vel = c->vel; f.part_ke = c->stage_a; f.hk = c->n3_hk; f.dt = c->n3_dt;
    if (f.fuse && !mixed) { f.xf = nullptr; f.xfr = nullptr; }
    if (f.fuse && mixed) { f.xf = c->xf; f.xfr = c->xfr; }
    const int fb = ceil_div(N, kN3FinAtoms);
    if (force) n3_finalize_kernel<true><<<fb, kN3FinWarps * 32, 0, c->stream>>>(f);
    else n3_finalize_kernel<false><<<fb, kN3FinWarps * 32, 0, c->stream>>>(f);
    c->launches += 2;
    if (!force) {
        c->emb_pending = fb;
    } else if (energy) {
        reduce_partials_kernel<<<1, 1024, 0, c->stream>>>(c->part_b, pieces, c->scal, kSlotEPair, c->consts.En);
        c->launches += 1;
    }
    SC_CUDA_CHECK(c, cudaGetLastError());
    return SC_OK;
}

// all pairs: do the sweeps run the Newton's-third-law kernels (sc_allpairs_n3.cuh) for this context as configured?
bool n3_wanted(const sc_ctx *c) {
    if (c->cutoff || !c->n3_part || c->opt_n3 == 2 || c->split) return false;
    return c->opt_n3 == 1 || (c->N >= (c->precision == SC_PREC_MIXED ? kN3DefaultMinAtomsMixed : kN3DefaultMinAtoms) &&
                              !c->opt_it && !c->opt_tpr);
}

sc_status run_sweep(sc_ctx *c, bool force, bool energy) {
    if (c->cutoff) return run_sweep_cutoff(c, force, energy);
    if (n3_wanted(c)) return run_sweep_n3(c, force, energy);
    TileChoice tc = choose_tile(c, force, energy);
    const void *fn = allpairs_fn(c, tc.it, tc.tpr, force, energy);
    if (!fn) return fail(c, SC_ERR_INVALID, "all-pairs sweep: no kernel for this tile shape%s");
    const int rpc = allpairs_rows_per_cta(tc.it, tc.tpr);
    const int grid = ceil_div(c->row_end - c->row_begin, rpc);
    const size_t smem = allpairs_smem_bytes(tc.it, tc.tpr, tc.warps);
    AllPairsArgs a{};
    a.xs = c->xs; a.n_atoms = int(c->N); a.row_begin = c->row_begin; a.row_end = c->row_end; a.rho = c->rho; a.force = c->force;
    a.partial = force ? c->part_b : c->part_a;
    a.c = c->consts;
    AllPairs32Args a32{};
    a32.xf = c->xf; a32.xs = c->xs; a32.n_atoms = a.n_atoms; a32.row_begin = a.row_begin; a32.row_end = a.row_end; a32.rho = a.rho; a32.force = a.force; a32.partial = a.partial;
    a32.c = c->consts;
    void *params[1] = {c->precision == SC_PREC_MIXED ? static_cast<void *>(&a32) : static_cast<void *>(&a)};
    cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem));
    if (e == cudaSuccess) e = cudaLaunchKernel(fn, dim3(grid), dim3((tc.warps + 1) * 32), params, smem, c->stream);
    if (e != cudaSuccess) return fail(c, SC_ERR_CUDA, "all-pairs sweep launch: %s", cudaGetErrorString(e));
    c->launches += 1;
    if (!force) {
        c->emb_pending = grid;
    } else if (energy) {
        reduce_partials_kernel<<<1, 1024, 0, c->stream>>>(a.partial, grid, c->scal, kSlotEPair, c->consts.En);
        SC_CUDA_CHECK(c, cudaGetLastError());
        c->launches += 1;
    }
    return SC_OK;
}

sc_status ensure_density(sc_ctx *c) {
    if (c->density_valid) return SC_OK;
    if (c->split) return fail(c, SC_ERR_STATE, "row split: densities come from the exchange; run sc_step_rows phases 1 and 2 first%s");
    sc_status st = run_sweep(c, false, false);
    if (st == SC_OK) c->density_valid = true;
    return st;
}

sc_status ensure_forces(sc_ctx *c, bool energy) {
    if (c->forces_valid && (!energy || c->energy_valid)) return SC_OK;
    if (c->split) return fail(c, SC_ERR_STATE, "row split: run sc_step_rows phases 1 and 2 to evaluate the forces%s");
    if (c->profile) cudaEventRecord(c->ev[0], c->stream);
    sc_status st = ensure_density(c);
    if (st != SC_OK) return st;
    if (energy && c->emb_pending) {
        // U_emb = -eps c sum sqrt(rho_i) from the per-CTA sums sweep 1 left behind: only energy steps pay for this launch
        reduce_partials_kernel<<<1, 1024, 0, c->stream>>>(c->part_a, c->emb_pending, c->scal, kSlotEEmb, -c->consts.eps_c);
        SC_CUDA_CHECK(c, cudaGetLastError());
        c->launches += 1;
        c->emb_pending = 0;
    }
    if (c->profile) cudaEventRecord(c->ev[1], c->stream);
    st = run_sweep(c, true, energy);
    if (st != SC_OK) return st;
    if (c->profile) cudaEventRecord(c->ev[2], c->stream);
    c->forces_valid = true;
    if (energy) c->energy_valid = true;
    return SC_OK;
}

sc_status flush_lambda(sc_ctx *c) {
    if (!c->lambda_pending) return SC_OK;
    const int n3 = int(3 * c->N);
    scale_velocities_kernel<<<ceil_div(n3, kBlock), kBlock, 0, c->stream>>>(c->vel, c->scal, n3);
    reset_lambda_kernel<<<1, 1, 0, c->stream>>>(c->scal);
    SC_CUDA_CHECK(c, cudaGetLastError());
    c->launches += 2;
    c->lambda_pending = false;
    return SC_OK;
}

sc_status read_scalars(sc_ctx *c, double *host, int count) {
    SC_CUDA_CHECK(c, cudaMemcpyAsync(host, c->scal, sizeof(double) * count, cudaMemcpyDeviceToHost, c->stream));
    SC_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    return SC_OK;
}

// internal array (internal atom order) -> caller's device buffer (caller's order), width doubles per atom
sc_status copy_out(sc_ctx *c, const double *src, double *d_dst, int width) {
    const int N = int(c->N);
    if (c->cutoff) {
        scatter_by_perm_kernel<<<ceil_div(N, kBlock), kBlock, 0, c->stream>>>(src, d_dst, c->perm, N, width);
        SC_CUDA_CHECK(c, cudaGetLastError());
        c->launches += 1;
    } else {
        SC_CUDA_CHECK(c, cudaMemcpyAsync(d_dst, src, sizeof(double) * size_t(width) * size_t(N), cudaMemcpyDeviceToDevice, c->stream));
    }
    return SC_OK;
}

// ---------------------------------------------------------------------------------------------
// one-launch step loop (sc_small.cuh): small all-pairs FP64 clusters
// ---------------------------------------------------------------------------------------------
// measured crossovers with the multi-launch path (Newton's-third-law sweeps, FP64; one-sided packed sweeps, mixed):
// FP64: N = 3000 43 us per step either way, N = 4096 62.5 (loop) against 61.5 us, N = 5000 129 against 68 us;
// mixed: N = 2057 23 (loop) against 28 us, N = 2500 44 against 37 us
// round 2, after the balanced plan and n3_loop_kernel (500-step NVE calls, us per step, one-launch loop of sc_small.cuh
// against the Newton's-third-law loop): FP64 N = 2057 20.5 / 24.3, 2304 22.0 / 24.7, 2560 37.5 / 24.5, 3072 43.9 / 30.5,
// 4096 62.2 / 39.0; mixed 2304 21.7 / 23.4, 2560 38.0 / 23.6, 3072 44.7 / 30.9.  After the lean terms, the conflict-free staged
// records and the free thread layout of the one-sided loop (1000-step calls): FP64 N = 2368 18.9 / 24.6, 2560 24.7 / 25.4,
// 2960 27.5 / 30.6, 3072 32.3 / 30.6; mixed 2368 17.8 / 23.4, 2960 25.7 / 30.4, 3552 33.5 / 31.4: up to 20 rows per CTA on 148 SMs
constexpr int64_t kSmallDefaultMaxAtoms = 2960, kSmallDefaultMaxAtomsMixed = 2960;

bool small_path_wanted(const sc_ctx *c) {
    if (c->cutoff || !c->xs_b || c->opt_persistent >= 2 || c->profile || c->split) return false;
    if (c->N > kSmallMaxAtoms) return false;
    if (ceil_div(c->N, c->sm_count) > (kSmallThreads / 32) * kSmallMaxRowsPerWarp) return false;   // no thread layout (a device with few SMs)
    return c->opt_persistent == 1 || c->N <= (c->precision == SC_PREC_MIXED ? kSmallDefaultMaxAtomsMixed : kSmallDefaultMaxAtoms);
}

sc_status run_small_steps(sc_ctx *c, double dt, const sc_thermostat *th, int thermo, int64_t nsteps) {
    const bool fast = (c->p.n == 9 && c->p.m == 6);
    const bool mixed = c->precision == SC_PREC_MIXED;
    const void *fn = mixed ? (fast ? reinterpret_cast<const void *>(small_step_kernel<9, 6, true>)
                                   : reinterpret_cast<const void *>(small_step_kernel<0, 0, true>))
                           : (fast ? reinterpret_cast<const void *>(small_step_kernel<9, 6, false>)
                                   : reinterpret_cast<const void *>(small_step_kernel<0, 0, false>));
    const int N = int(c->N);
    const size_t smem = small_step_smem_bytes(N);
    if (c->small_ctas == 0) {
        int per_sm = 0;
        SC_CUDA_CHECK(c, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem)));
        SC_CUDA_CHECK(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, kSmallThreads, smem));
        if (per_sm < 1) return fail(c, SC_ERR_CUDA, "one-launch step loop: kernel does not fit on an SM%s");
        c->small_ctas = c->sm_count;                    // one CTA per SM: the barrier cost grows with the CTA count
    }
    SmallStepArgs a{};
    a.xs = c->xs; a.xs_b = c->xs_b; a.xf = c->xf; a.xfr = c->xfr; a.vel = c->vel; a.force = c->force; a.rho = c->rho;
    a.part_emb = c->part_a; a.part_pair = c->part_b; a.part_ke = c->part_ke; a.scal = c->scal;
    a.sprime = c->sprime; a.barrier = c->small_barrier; a.barrier_base = c->small_barrier_count;
    a.n_atoms = N;
    a.rows = ceil_div(N, c->small_ctas);
    const int grid = ceil_div(N, a.rows);
    // Thread layout: a warp holds rpw = 1, 2, 4 or 8 rows (lq = 32 / rpw lanes each; more rows per warp = fewer
    // shared-memory wavefronts per pair), a row group of rpw rows is spread over wpg warps (ANY count, not a power of two:
    // jl = lq x wpg threads stride the j range of a row), and the groups x wpg warps share the SM's four sub-partitions.
    // The sweeps last (warps of the busiest sub-partition) x (pairs per thread); the host takes the layout that makes
    // that product smallest, the larger rpw on a tie.  (Round 1 took jl as a power of two: N = 1415 -- 10 rows per CTA --
    // ran 10 warps of 44 pairs per thread, 2 - 3 per sub-partition, too few to hide the FP64 latency: sweeps of 4.0 + 4.7 us
    // where 15 warps of 30 pairs take 2.9 + 3.6.)
    int best_rpw = 1, best_wpg = 1;
    double best_cost = 0.0;
    const int forced = c->opt_tpr ? std::min(32 / c->opt_tpr, kSmallMaxRowsPerWarp) : 0;   // SC_OPT_LANES_PER_ROW
    for (int pass = 0; pass < 2 && best_cost == 0.0; ++pass)       // second pass: the forced layout does not fit
        for (int rpw : {8, 4, 2, 1}) {
            if (pass == 0 && forced && rpw != forced) continue;
            const int groups = ceil_div(a.rows, rpw);
            int wpg = (kSmallThreads / 32) / groups;
            if (rpw == 8) wpg &= ~1;                                // jl = lq x wpg must be a multiple of 8 (small_rec_off)
            if (wpg < 1) continue;
            const int jl_c = (32 / rpw) * wpg, warps = groups * wpg;
            // a row that lives in ONE warp (wpg = 1) needs no pass through shared memory and no CTA barriers for its sums:
            // measured 2 - 10 % per step where it ties on the product (N = 1776 15.2 -> 13.7 us, 2057 16.8 -> 16.45, mixed 16.1 -> 15.3)
            const double cost = double(ceil_div(warps, 4)) * double(ceil_div(N, jl_c)) * (wpg == 1 ? 0.97 : 1.0);
            if (best_cost == 0.0 || cost < best_cost - 1e-9) { best_cost = cost; best_rpw = rpw; best_wpg = wpg; }
        }
    if (best_cost == 0.0) return fail(c, SC_ERR_INVALID, "one-launch step loop: no thread layout for this size%s");
    a.lq = 32 / best_rpw;
    a.jl = a.lq * best_wpg;
    if (32 / a.lq > kSmallMaxRowsPerWarp) return fail(c, SC_ERR_INVALID, "one-launch step loop: more than 8 rows per warp%s");
    a.nsteps = nsteps; a.hk = 0.5 * dt * kAcc / c->p.mass; a.dt = dt; a.mass = c->p.mass; a.ndof = double(3 * c->N - 3);
    a.thermo = thermo;
    if (th) { a.T_start = th->T_start; a.T_end = th->T_end; }
    if (thermo == SC_THERMO_LANGEVIN) {
        a.lg_c1 = std::exp(-th->gamma * dt);
        a.lg_pre = (1.0 - a.lg_c1 * a.lg_c1) * kBoltzmann;
        a.key0 = uint32_t(th->seed); a.key1 = uint32_t(th->seed >> 32);
        a.lg_step0 = c->langevin_step;
    }
    a.c = c->consts;
    void *params[] = {&a};
    cudaError_t e = cudaLaunchCooperativeKernel(fn, dim3(grid), dim3(kSmallThreads), params, smem, c->stream);
    if (e != cudaSuccess) return fail(c, SC_ERR_CUDA, "one-launch step loop: %s", cudaGetErrorString(e));
    c->launches += 1;
    // barriers of this launch: 2 per step, a third on rescale steps and on the last step, one in the epilogue
    const uint64_t nbar = 2 * uint64_t(nsteps) + (thermo == SC_THERMO_RESCALE ? uint64_t(nsteps) : 1) + 1;
    c->small_barrier_count += nbar * uint64_t(grid);
    if (thermo == SC_THERMO_LANGEVIN) c->langevin_step += uint64_t(nsteps);
    c->lambda_pending = false;                           // consumed (and the last scale applied) by the kernel
    c->emb_pending = 0;                                  // the loop wrote both energy scalars itself
    c->density_valid = c->forces_valid = c->energy_valid = true;
    return SC_OK;
}

// ---------------------------------------------------------------------------------------------
// NVE steps through the Newton's-third-law sweeps in one cooperative launch (sc_n3_loop.cuh)
// ---------------------------------------------------------------------------------------------
// Measured against the four launches per step (300-step calls, us per step): N = 4096 39.0 / 45.1, N = 8000 100.2 / 103.1,
// mixed 82.6 / 87.9, N = 16384 353.7 / 352.6, N = 32768 1373 / 1328: beyond ~12000 atoms the finalize phases, which read
// N^2 / 512 partial records with 8 warps per SM, cost more than the stand-alone finalize kernels (64 warps per SM) save.
// After the pair blocks (finalize phases read half as much): N = 12288 196.8 / 200.4, 14336 262.0 / 264.7, 16384 337.5 / 337.9,
// 20480 520.7 / 510.4; mixed 16384 248.3 / 250.0, 20480 381.4 / 373.0.
constexpr int64_t kN3LoopMaxAtoms = 16384;

bool n3_loop_wanted(const sc_ctx *c, int thermo) {
    return (thermo == SC_THERMO_NONE || thermo == SC_THERMO_RESCALE) && n3_wanted(c) && !c->profile && c->opt_persistent != 2 && c->n3_barrier &&
           c->N <= kN3LoopMaxAtoms && !(c->opt_warps && c->opt_warps <= 6) && c->opt_n3_pieces >= 0 && c->opt_n3_pieces <= 1;
}

// positions already carry the first half kick + drift of the call's first step (kick_drift_kernel)
sc_status run_n3_loop(sc_ctx *c, double dt, const sc_thermostat *th, int thermo, int64_t nsteps) {
    const bool fast = (c->p.n == 9 && c->p.m == 6), mixed = c->precision == SC_PREC_MIXED;
    const int N = int(c->N), rb = kN3PairRows;
    if (!c->n3_seg) {
        sc_status st = plan_n3(c);
        if (st != SC_OK) return st;
    }
    const int pieces = c->n3_seg;
    const void *fn = n3_loop_fn(fast, mixed);
    N3LoopArgs a{};
    a.s.xs = c->xs; a.s.n_atoms = N; a.s.n_pad = round_up(N, 32);
    a.s.part = c->n3_part; a.s.part_rho = reinterpret_cast<double *>(c->n3_part); a.s.self = c->n3_self;
    a.s.partial = c->part_b; a.s.tiles = c->n3_tiles; a.s.piece_start = c->n3_piece_start; a.s.c = c->consts;
    a.sf.xfr = c->xfr; a.sf.n_atoms = N; a.sf.n_pad = a.s.n_pad; a.sf.part = a.s.part; a.sf.part_rho = a.s.part_rho;
    a.sf.self = a.s.self; a.sf.partial = a.s.partial; a.sf.tiles = a.s.tiles; a.sf.piece_start = a.s.piece_start; a.sf.c = a.s.c;
    N3FinalArgs &f = a.f;
    f.xs = c->xs; f.xfr = mixed ? c->xfr : nullptr; f.xf = mixed ? c->xf : nullptr; f.part = c->n3_part; f.part_rho = a.s.part_rho;
    f.self = c->n3_self; f.rho = c->rho; f.force = c->force; f.partial = c->part_a; f.n_atoms = N; f.n_pad = a.s.n_pad; f.rb = rb;
    f.blk_slots = c->n3_blk_slots; f.c = c->consts; f.fuse = 0; f.vel = c->vel; f.part_ke = c->stage_a;
    f.hk = 0.5 * dt * kAcc / c->p.mass; f.dt = dt;
    a.barrier = c->n3_barrier; a.barrier_base = c->n3_barrier_count;
    a.nsteps = nsteps; a.energy_every = c->opt_energy_every;
    a.thermo = thermo == SC_THERMO_RESCALE ? 1 : 0;
    a.mass = c->p.mass; a.ndof = double(3 * c->N - 3);
    if (th) { a.T_start = th->T_start; a.T_end = th->T_end; }
    void *params[] = {&a};
    cudaError_t e = cudaLaunchCooperativeKernel(fn, dim3(pieces), dim3(kN3Warps * 32), params, 0, c->stream);
    if (e != cudaSuccess) return fail(c, SC_ERR_CUDA, "Newton's-third-law step loop: %s", cudaGetErrorString(e));
    c->launches += 1;
    c->n3_barrier_count += (4 * uint64_t(nsteps) - 1 + (a.thermo ? uint64_t(nsteps) - 1 : 0)) * uint64_t(pieces);
    const int nfin = ceil_div(N, kN3FinAtoms);
    reduce_partials_kernel<<<1, 1024, 0, c->stream>>>(c->part_b, pieces, c->scal, kSlotEPair, c->consts.En);
    reduce_partials_kernel<<<1, 1024, 0, c->stream>>>(c->part_a, nfin, c->scal, kSlotEEmb, -c->consts.eps_c);
    // KE and T of the last step; rescaling: its lambda is left pending as on the other paths (flush_lambda)
    reduce_ke_kernel<<<1, 1024, 0, c->stream>>>(c->stage_a, nfin, c->scal, c->p.mass, a.ndof, thermo,
                                             a.thermo ? a.T_start + (a.T_end - a.T_start) * double(nsteps) / double(nsteps) : 0.0);
    if (a.thermo) c->lambda_pending = true;
    SC_CUDA_CHECK(c, cudaGetLastError());
    c->launches += 3;
    c->emb_pending = 0;
    c->density_valid = c->forces_valid = c->energy_valid = true;
    return SC_OK;
}

sc_status do_step(sc_ctx *c, double dt, const sc_thermostat *th, int64_t nsteps) {
    if (!c->have_pos || !c->have_vel) return fail(c, SC_ERR_STATE, "sc_step: positions and velocities must be set%s");
    if (!(dt > 0.0) || !std::isfinite(dt) || nsteps < 0) return fail(c, SC_ERR_INVALID, "sc_step: dt must be > 0, nsteps >= 0%s");
    int thermo = SC_THERMO_NONE;
    if (th) {
        thermo = th->kind;
        if (thermo != SC_THERMO_NONE && thermo != SC_THERMO_RESCALE && thermo != SC_THERMO_LANGEVIN)
            return fail(c, SC_ERR_INVALID, "sc_step: unknown thermostat kind%s");
        if (thermo != SC_THERMO_NONE && !(th->T_start >= 0.0 && th->T_end >= 0.0 && std::isfinite(th->T_start) && std::isfinite(th->T_end)))
            return fail(c, SC_ERR_INVALID, "sc_step: thermostat temperatures must be finite and >= 0%s");
        if (thermo == SC_THERMO_LANGEVIN && !(th->gamma >= 0.0 && std::isfinite(th->gamma)))
            return fail(c, SC_ERR_INVALID, "sc_step: Langevin damping must be finite and >= 0 (1/fs)%s");
    }
    if (nsteps == 0) return SC_OK;
    if (c->split) return fail(c, SC_ERR_STATE, "sc_step: this context is one rank of a row split; use sc_step_rows%s");
    sc_status st = ensure_forces(c, false);
    if (st != SC_OK) return st;
    if (small_path_wanted(c)) return run_small_steps(c, dt, th, thermo, nsteps);
    const int N = int(c->N);
    const int nb = ceil_div(N, kBlock);
    const double hk = 0.5 * dt * kAcc / c->p.mass;
    const double ndof = double(3 * c->N - 3);
    // NVE steps through the Newton's-third-law sweeps: the force finalize kernel does the second half kick and (except on
    // the last step) the first half kick and the drift of the next step: 4 launches per step instead of 6
    const bool fused = thermo == SC_THERMO_NONE && n3_wanted(c) && !c->profile;
    const int nfin = ceil_div(N, kN3FinAtoms);
    if (n3_loop_wanted(c, thermo)) {
        kick_drift_kernel<<<nb, kBlock, 0, c->stream>>>(c->xs, c->vel, c->force, c->scal, nullptr, c->xf, c->xfr, 0, N, hk, dt);
        SC_CUDA_CHECK(c, cudaGetLastError());
        c->launches += 1;
        c->density_valid = c->forces_valid = c->energy_valid = false;
        st = run_n3_loop(c, dt, th, thermo, nsteps);
        if (st != SC_OK) return st;
        return flush_lambda(c);
    }
    for (int64_t k = 1; k <= nsteps; ++k) {
        const bool last = (k == nsteps);
        if (!fused || k == 1) {
            kick_drift_kernel<<<nb, kBlock, 0, c->stream>>>(c->xs, c->vel, c->force, c->scal, c->cutoff ? c->xs_ref : nullptr,
                                                            c->xf, c->xfr, 0, N, hk, dt);
            SC_CUDA_CHECK(c, cudaGetLastError());
            c->launches += 1;
        }
        c->density_valid = c->forces_valid = c->energy_valid = false;
        c->list_checked = false;
        c->n3_fuse = fused ? (last ? 1 : 2) : 0; c->n3_hk = hk; c->n3_dt = dt;
        st = ensure_forces(c, last || c->opt_energy_every == 1);
        c->n3_fuse = 0;
        if (st != SC_OK) return st;
        if (fused) {
            if (last) {
                reduce_ke_kernel<<<1, 1024, 0, c->stream>>>(c->stage_a, nfin, c->scal, c->p.mass, ndof, thermo, 0.0);
                c->launches += 1;
            }
            SC_CUDA_CHECK(c, cudaGetLastError());
            continue;
        }
        if (thermo == SC_THERMO_LANGEVIN) {
            const double target = th->T_start + (th->T_end - th->T_start) * double(k) / double(nsteps);
            LangevinArgs lg{};
            lg.c1 = std::exp(-th->gamma * dt);
            lg.c2 = std::sqrt((1.0 - lg.c1 * lg.c1) * kBoltzmann * target * kAcc / c->p.mass);
            lg.key0 = uint32_t(th->seed); lg.key1 = uint32_t(th->seed >> 32);
            lg.step_lo = uint32_t(c->langevin_step); lg.step_hi = uint32_t(c->langevin_step >> 32);
            lg.perm = c->cutoff ? c->perm : nullptr;
            kick_langevin_ke_kernel<<<nb, kBlock, 0, c->stream>>>(c->vel, c->force, c->part_ke, 0, N, hk, lg);
            c->langevin_step += 1;
        } else {
            kick_ke_kernel<<<nb, kBlock, 0, c->stream>>>(c->vel, c->force, c->part_ke, 0, N, hk);
        }
        c->launches += 1;
        if (thermo == SC_THERMO_RESCALE || last) {
            const double target = thermo == SC_THERMO_RESCALE
                                      ? th->T_start + (th->T_end - th->T_start) * double(k) / double(nsteps)
                                      : 0.0;
            reduce_ke_kernel<<<1, 1024, 0, c->stream>>>(c->part_ke, nb, c->scal, c->p.mass, ndof, thermo, target);
            c->launches += 1;
            if (thermo == SC_THERMO_RESCALE) c->lambda_pending = true;
        }
        SC_CUDA_CHECK(c, cudaGetLastError());       // the integrator launches of this step
    }
    sc_status fl = flush_lambda(c);
    if (fl != SC_OK) return fl;
    return check_flags(c);          // cutoff path only: one synchronisation per sc_step call
}

}  // namespace

// =============================================================================================
// C ABI
// =============================================================================================
extern "C" {

const char *sc_version(void) { return "libscmd 0.1 (sm_100a)"; }

const char *sc_last_error(const sc_ctx *ctx) { return ctx ? ctx->err : "null context"; }

size_t sc_workspace_bytes_ex(const sc_params *params, int64_t n_atoms, int32_t precision, double skin,
                             const sc_create_options *options) {
    if (!params_ok(params) || n_atoms < 1 || n_atoms > (int64_t(1) << 30)) return 0;
    if (precision != SC_PREC_FP64 && precision != SC_PREC_MIXED) return 0;
    if (!(skin >= 0.0) || !create_options_ok(options)) return 0;
    if (params->r_cut > 0.0 && n_atoms > kCutoffMaxAtoms) return 0;       // run words hold 29-bit indices
    if (row_split(options) && (params->r_cut > 0.0 || options->row_end > n_atoms)) return 0;   // the row split is all pairs only
    return carve(nullptr, nullptr, n_atoms, params, precision, skin, options);
}

size_t sc_workspace_bytes(const sc_params *params, int64_t n_atoms, int32_t precision, double skin) {
    return sc_workspace_bytes_ex(params, n_atoms, precision, skin, nullptr);
}

sc_status sc_create(const sc_params *params, int64_t n_atoms, int32_t precision, double skin, void *d_workspace,
                    size_t workspace_bytes, void *cuda_stream, sc_ctx **out) {
    return sc_create_ex(params, n_atoms, precision, skin, nullptr, d_workspace, workspace_bytes, cuda_stream, out);
}

sc_status sc_create_ex(const sc_params *params, int64_t n_atoms, int32_t precision, double skin,
                       const sc_create_options *options, void *d_workspace, size_t workspace_bytes, void *cuda_stream,
                       sc_ctx **out) {
    if (!out) return SC_ERR_INVALID;
    *out = nullptr;
    if (!params_ok(params) || n_atoms < 1 || n_atoms > (int64_t(1) << 30)) return SC_ERR_INVALID;
    if (precision != SC_PREC_FP64 && precision != SC_PREC_MIXED) return SC_ERR_INVALID;
    if (!(skin >= 0.0) || !d_workspace || !create_options_ok(options)) return SC_ERR_INVALID;
    if (reinterpret_cast<uintptr_t>(d_workspace) % kAlign) return SC_ERR_INVALID;
    if (params->r_cut > 0.0 && n_atoms > kCutoffMaxAtoms) return SC_ERR_INVALID;
    if (row_split(options) && (params->r_cut > 0.0 || options->row_end > n_atoms)) return SC_ERR_INVALID;
    const size_t need = sc_workspace_bytes_ex(params, n_atoms, precision, skin, options);
    if (workspace_bytes < need) return SC_ERR_NOMEM;
    int dev = 0, count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || count < 1) return SC_ERR_CUDA;
    if (cudaGetDevice(&dev) != cudaSuccess) return SC_ERR_CUDA;
    sc_ctx *c = new (std::nothrow) sc_ctx();
    if (!c) return SC_ERR_NOMEM;
    c->p = *params; c->N = n_atoms; c->precision = precision; c->skin = skin;
    c->row_begin = 0; c->row_end = int(n_atoms);
    if (row_split(options)) { c->split = true; c->row_begin = options->row_begin; c->row_end = options->row_end; }
    c->stream = static_cast<cudaStream_t>(cuda_stream);
    cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, dev);
    carve(c, d_workspace, n_atoms, params, precision, skin, options);
    const double a_n = ipow_host(params->a, params->n), a_m = ipow_host(params->a, params->m);
    c->consts.am = a_m;
    c->consts.An = params->eps * params->n * a_n;
    c->consts.Bm = params->eps * (params->c * params->m / 2.0) * a_m;
    c->consts.En = params->eps / 2.0 * a_n;
    c->consts.eps_c = params->eps * params->c;
    c->consts.n = params->n; c->consts.m = params->m;
    for (auto &e : c->ev)
        if (cudaEventCreate(&e) != cudaSuccess) { delete c; return SC_ERR_CUDA; }
    // scalars: zero, lambda = 1; pad the record array tail so that full-tile reads stay defined
    if (cudaMemsetAsync(c->scal, 0, sizeof(double) * kNumScalars, c->stream) != cudaSuccess ||
        cudaMemsetAsync(c->xs, 0, sizeof(double4) * (size_t(n_atoms) + kTileAtoms), c->stream) != cudaSuccess ||
        (c->xf && cudaMemsetAsync(c->xf, 0, sizeof(FPair) * ((size_t(n_atoms) + kTileAtoms) / 2 + 1), c->stream) != cudaSuccess)) {
        delete c;
        return SC_ERR_CUDA;
    }
    reset_lambda_kernel<<<1, 1, 0, c->stream>>>(c->scal);
    if (cudaGetLastError() != cudaSuccess) { delete c; return SC_ERR_CUDA; }
    if (c->n3_barrier && cudaMemsetAsync(c->n3_barrier, 0, 2 * sizeof(unsigned long long), c->stream) != cudaSuccess) {
        delete c;
        return SC_ERR_CUDA;
    }
    if (c->small_barrier && cudaMemsetAsync(c->small_barrier, 0, 2 * sizeof(unsigned long long), c->stream) != cudaSuccess) {
        delete c;
        return SC_ERR_CUDA;
    }
    if (params->r_cut > 0.0) {
        c->cutoff = true;
        c->r_list = params->r_cut + skin;
        int per_sm = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, rebuild_kernel, 256, 0) != cudaSuccess || per_sm < 1) {
            delete c;
            return SC_ERR_CUDA;
        }
        if (per_sm > 4) per_sm = 4;
        c->coop_grid = per_sm * c->sm_count;
        const int want = ceil_div(n_atoms, 16);             // neighbour rows are built one warp per atom pair
        if (c->coop_grid > want) c->coop_grid = want;
        if (c->coop_grid > kMaxCoopBlocks) c->coop_grid = kMaxCoopBlocks;
        if (cudaMemsetAsync(c->counters, 0, sizeof(unsigned long long) * kNumCounters, c->stream) != cudaSuccess ||
            cudaMemsetAsync(c->xs_alt, 0, sizeof(double4) * (size_t(n_atoms) + kTileAtoms), c->stream) != cudaSuccess) {
            delete c;
            return SC_ERR_CUDA;
        }
        iota_kernel<<<ceil_div(n_atoms, kBlock), kBlock, 0, c->stream>>>(c->perm, int(n_atoms));
        if (cudaGetLastError() != cudaSuccess) { delete c; return SC_ERR_CUDA; }
    }
    *out = c;
    return SC_OK;
}

sc_status sc_destroy(sc_ctx *ctx) {
    if (!ctx) return SC_ERR_INVALID;
    cudaStreamSynchronize(ctx->stream);
    for (auto &e : ctx->ev)
        if (e) cudaEventDestroy(e);
    delete ctx;
    return SC_OK;
}

sc_status sc_set_option(sc_ctx *c, int32_t option, int64_t value) {
    if (!c) return SC_ERR_INVALID;
    auto pow2_le32 = [](int64_t v) { return v == 1 || v == 2 || v == 4 || v == 8 || v == 16 || v == 32; };
    switch (option) {
        case SC_OPT_ROWS_PER_THREAD:
            if (value != 0 && value != 1 && value != 2 && value != 4) return fail(c, SC_ERR_INVALID, "rows per thread must be 0, 1, 2 or 4%s");
            c->opt_it = int(value); break;
        case SC_OPT_LANES_PER_ROW:
            if (value != 0 && !pow2_le32(value)) return fail(c, SC_ERR_INVALID, "lanes per row must be a power of two <= 32%s");
            c->opt_tpr = int(value); break;
        case SC_OPT_WARPS_PER_CTA:
            if (value < 0 || value > (c->cutoff ? kNlistMaxBlock / 32 : kMaxConsumerWarps))
                return fail(c, SC_ERR_INVALID, "warps per CTA must be 0..8%s");
            c->opt_warps = int(value); c->n3_seg = 0; break;
        case SC_OPT_PERSISTENT:
            if (value < 0 || value > 3) return fail(c, SC_ERR_INVALID, "persistent must be 0, 1, 2 or 3%s");
            c->opt_persistent = int(value); break;
        case SC_OPT_ENERGY_EVERY_STEP:
            c->opt_energy_every = value ? 1 : 0; break;
        case SC_OPT_NEIGHBOUR_CAPACITY:
            if (value < 0 || (c->cutoff && value > c->kmax_cap))
                return fail(c, SC_ERR_INVALID, "neighbour capacity must be 0 .. the capacity the workspace was sized for%s");
            c->opt_kmax = int(value);
            if (c->cutoff) {
                c->kmax = value ? (value < 32 ? 32 : int(value) / 32 * 32) : c->kmax_cap;   // rows are padded to 32
                c->list_checked = false;
                reset_list_state_kernel<<<1, 1, 0, c->stream>>>(c->counters, c->scal);
                SC_CUDA_CHECK(c, cudaGetLastError());
                c->launches += 1;
                c->density_valid = c->forces_valid = c->energy_valid = false;
            }
            break;
        case SC_OPT_LANGEVIN_STEP:
            if (value < 0) return fail(c, SC_ERR_INVALID, "Langevin generator step must be >= 0%s");
            c->langevin_step = uint64_t(value); break;
        case SC_OPT_CELLS_PER_RADIUS:
            if (value < 0 || value > kFineMax) return fail(c, SC_ERR_INVALID, "cells per list radius must be 0..4%s");
            c->opt_fine = int(value);
            if (c->cutoff) {
                c->list_checked = false;
                reset_list_state_kernel<<<1, 1, 0, c->stream>>>(c->counters, c->scal);
                SC_CUDA_CHECK(c, cudaGetLastError());
                c->launches += 1;
                c->density_valid = c->forces_valid = c->energy_valid = false;
            }
            break;
        case SC_OPT_NEWTON3:
            if (value < 0 || value > 2) return fail(c, SC_ERR_INVALID, "Newton's third law must be 0, 1 or 2%s");
            c->opt_n3 = int(value);
            c->density_valid = c->forces_valid = c->energy_valid = false;
            break;
        case SC_OPT_CUTOFF_SHIFT:
            if (value < 0 || value > 1) return fail(c, SC_ERR_INVALID, "cutoff shift must be 0 or 1%s");
            c->opt_shift = int(value);
            c->density_valid = c->forces_valid = c->energy_valid = false;
            break;
        case SC_OPT_ATOMS_PER_CTA:
            if (value < 0 || value > 4096) return fail(c, SC_ERR_INVALID, "atoms per CTA must be 0..4096%s");
            c->opt_apc = int(value); break;
        case SC_OPT_NEWTON3_PIECES:
            if (value < -1 || value > 16) return fail(c, SC_ERR_INVALID, "Newton's-third-law pieces per SM must be -1..16%s");
            c->opt_n3_pieces = int(value); c->n3_seg = 0;
            c->density_valid = c->forces_valid = c->energy_valid = false;
            break;
        default:
            return fail(c, SC_ERR_INVALID, "unknown option%s");
    }
    if (c->opt_it == 4 && c->opt_tpr > 4) return fail(c, SC_ERR_INVALID, "4 rows per thread needs lanes per row <= 4%s");
    return SC_OK;
}

sc_status sc_get_option(sc_ctx *c, int32_t option, int64_t *value) {
    if (!c || !value) return fail(c, SC_ERR_INVALID, "sc_get_option: NULL argument%s");
    switch (option) {
        case SC_OPT_ROWS_PER_THREAD: *value = c->opt_it; break;
        case SC_OPT_LANES_PER_ROW: *value = c->opt_tpr; break;
        case SC_OPT_WARPS_PER_CTA: *value = c->opt_warps; break;
        case SC_OPT_PERSISTENT: *value = c->opt_persistent; break;
        case SC_OPT_ENERGY_EVERY_STEP: *value = c->opt_energy_every; break;
        case SC_OPT_NEIGHBOUR_CAPACITY: *value = c->opt_kmax; break;
        case SC_OPT_LANGEVIN_STEP: *value = int64_t(c->langevin_step); break;
        case SC_OPT_CELLS_PER_RADIUS: *value = c->opt_fine; break;
        case SC_OPT_ATOMS_PER_CTA: *value = c->opt_apc; break;
        case SC_OPT_NEWTON3: *value = c->opt_n3; break;
        case SC_OPT_CUTOFF_SHIFT: *value = c->opt_shift; break;
        case SC_OPT_NEWTON3_PIECES: *value = c->opt_n3_pieces; break;
        case SC_INFO_STEP_PATH:
            *value = c->cutoff ? 3 : (small_path_wanted(c) ? 2 : (n3_wanted(c) ? 1 : 0));
            break;
        case SC_INFO_NEIGHBOUR_CAPACITY: *value = c->cutoff ? c->kmax : 0; break;
        case SC_INFO_NEIGHBOUR_CAPACITY_MAX: *value = c->cutoff ? c->kmax_cap : 0; break;
        case SC_INFO_ONE_LAUNCH: *value = (small_path_wanted(c) || n3_loop_wanted(c, SC_THERMO_NONE)) ? 1 : 0; break;
        default:
            return fail(c, SC_ERR_INVALID, "sc_get_option: unknown option%s");
    }
    return SC_OK;
}

sc_status sc_set_state(sc_ctx *c, const double *d_pos, const double *d_vel) {
    if (!c || !d_pos) return fail(c, SC_ERR_INVALID, "sc_set_state: d_pos is NULL%s");
    const int N = int(c->N);
    pack_positions_kernel<<<ceil_div(N, kBlock), kBlock, 0, c->stream>>>(d_pos, c->xs, c->xf, c->xfr, N);
    SC_CUDA_CHECK(c, cudaGetLastError());
    c->launches += 1;
    c->have_pos = true;
    c->density_valid = c->forces_valid = c->energy_valid = false;
    if (c->cutoff) {
        // the internal order falls back to the caller's order; velocities already held follow it
        if (c->have_vel && !d_vel) {
            sc_status st = flush_lambda(c);
            if (st != SC_OK) return st;
            scatter_by_perm_kernel<<<ceil_div(N, kBlock), kBlock, 0, c->stream>>>(c->vel, c->vel_alt, c->perm, N, 3);
            SC_CUDA_CHECK(c, cudaMemcpyAsync(c->vel, c->vel_alt, sizeof(double) * 3 * size_t(N), cudaMemcpyDeviceToDevice, c->stream));
            c->launches += 1;
        }
        iota_kernel<<<ceil_div(N, kBlock), kBlock, 0, c->stream>>>(c->perm, N);
        reset_list_state_kernel<<<1, 1, 0, c->stream>>>(c->counters, c->scal);
        SC_CUDA_CHECK(c, cudaGetLastError());
        c->launches += 2;
        c->list_checked = false;
    }
    if (d_vel) {
        sc_status st = flush_lambda(c);
        if (st != SC_OK) return st;
        SC_CUDA_CHECK(c, cudaMemcpyAsync(c->vel, d_vel, sizeof(double) * 3 * size_t(N), cudaMemcpyDeviceToDevice, c->stream));
        c->have_vel = true;
    }
    return SC_OK;
}

sc_status sc_get_state(sc_ctx *c, double *d_pos, double *d_vel) {
    if (!c) return SC_ERR_INVALID;
    if (!c->have_pos) return fail(c, SC_ERR_STATE, "sc_get_state: no positions set%s");
    const int N = int(c->N);
    if (d_pos) {
        if (c->cutoff) unpack_positions_perm_kernel<<<ceil_div(N, kBlock), kBlock, 0, c->stream>>>(c->xs, d_pos, c->perm, N);
        else unpack_positions_kernel<<<ceil_div(N, kBlock), kBlock, 0, c->stream>>>(c->xs, d_pos, N);
        SC_CUDA_CHECK(c, cudaGetLastError());
        c->launches += 1;
    }
    if (d_vel) {
        if (!c->have_vel) return fail(c, SC_ERR_STATE, "sc_get_state: no velocities set%s");
        sc_status st = flush_lambda(c);
        if (st != SC_OK) return st;
        st = copy_out(c, c->vel, d_vel, 3);
        if (st != SC_OK) return st;
    }
    return SC_OK;
}

sc_status sc_density(sc_ctx *c, double *d_rho) {
    if (!c || !d_rho) return fail(c, SC_ERR_INVALID, "sc_density: NULL argument%s");
    if (!c->have_pos) return fail(c, SC_ERR_STATE, "sc_density: no positions set%s");
    sc_status st = ensure_density(c);
    if (st != SC_OK) return st;
    return copy_out(c, c->rho, d_rho, 1);
}

sc_status sc_forces(sc_ctx *c, double *d_force) {
    if (!c || !d_force) return fail(c, SC_ERR_INVALID, "sc_forces: NULL argument%s");
    if (!c->have_pos) return fail(c, SC_ERR_STATE, "sc_forces: no positions set%s");
    sc_status st = ensure_forces(c, true);
    if (st != SC_OK) return st;
    return copy_out(c, c->force, d_force, 3);
}

sc_status sc_energy(sc_ctx *c, double *h_epot) {
    if (!c || !h_epot) return fail(c, SC_ERR_INVALID, "sc_energy: NULL argument%s");
    if (!c->have_pos) return fail(c, SC_ERR_STATE, "sc_energy: no positions set%s");
    if (!c->energy_valid) { c->forces_valid = false; }
    sc_status st = ensure_forces(c, true);
    if (st != SC_OK) return st;
    double s[2];
    st = read_scalars(c, s, 2);
    if (st != SC_OK) return st;
    *h_epot = s[kSlotEPair] + s[kSlotEEmb];
    if (!std::isfinite(*h_epot)) return fail(c, SC_ERR_NONFINITE, "sc_energy: potential energy is not finite (coincident atoms?)%s");
    return check_flags(c);
}

sc_status sc_kinetic(sc_ctx *c, double *h_ke, double *h_temperature) {
    if (!c || (!h_ke && !h_temperature)) return fail(c, SC_ERR_INVALID, "sc_kinetic: NULL argument%s");
    if (!c->have_vel) return fail(c, SC_ERR_STATE, "sc_kinetic: no velocities set%s");
    sc_status st = flush_lambda(c);
    if (st != SC_OK) return st;
    // one rank of a row split: its own atoms' share of the kinetic energy; T is then the caller's arithmetic on the sum
    const int nb = ceil_div(c->row_end - c->row_begin, kBlock);
    sum_v2_kernel<<<nb, kBlock, 0, c->stream>>>(c->vel, c->part_ke, c->row_begin, c->row_end, 0.0, c->scal);
    reduce_ke_kernel<<<1, 1024, 0, c->stream>>>(c->part_ke, nb, c->scal, c->p.mass, c->split ? 0.0 : double(3 * c->N - 3), 0, 0.0);
    SC_CUDA_CHECK(c, cudaGetLastError());
    c->launches += 2;
    double s[kSlotTemp + 1];
    st = read_scalars(c, s, kSlotTemp + 1);
    if (st != SC_OK) return st;
    if (h_ke) *h_ke = s[kSlotKE];
    if (h_temperature) *h_temperature = s[kSlotTemp];
    if (!std::isfinite(s[kSlotKE])) return fail(c, SC_ERR_NONFINITE, "sc_kinetic: kinetic energy is not finite%s");
    return SC_OK;
}

sc_status sc_step(sc_ctx *c, double dt_fs, const sc_thermostat *thermostat, int64_t nsteps) {
    if (!c) return SC_ERR_INVALID;
    return do_step(c, dt_fs, thermostat, nsteps);
}

sc_status sc_step_rows(sc_ctx *c, int32_t phase, double dt, const sc_thermostat *th, double *d_pos_all, double *d_rho_all) {
    if (!c) return SC_ERR_INVALID;
    if (!c->split) return fail(c, SC_ERR_STATE, "sc_step_rows: the context was not created as a rank of a row split%s");
    if (phase < 0 || phase > 2 || !(dt >= 0.0) || !std::isfinite(dt))
        return fail(c, SC_ERR_INVALID, "sc_step_rows: phase must be 0, 1 or 2 and dt >= 0%s");
    if (!c->have_pos) return fail(c, SC_ERR_STATE, "sc_step_rows: no positions set%s");
    int thermo = th ? th->kind : SC_THERMO_NONE;
    if (thermo != SC_THERMO_NONE && thermo != SC_THERMO_LANGEVIN)
        return fail(c, SC_ERR_INVALID, "sc_step_rows: only NVE and the Langevin thermostat work rank by rank%s");
    if (thermo == SC_THERMO_LANGEVIN && !(th->gamma >= 0.0 && std::isfinite(th->gamma) && th->T_end >= 0.0 && std::isfinite(th->T_end)))
        return fail(c, SC_ERR_INVALID, "sc_step_rows: Langevin damping and temperature must be finite and >= 0%s");
    const int N = int(c->N), rb = c->row_begin, re = c->row_end, rows = re - rb;
    const int nb_rows = ceil_div(rows, kBlock), nb_all = ceil_div(N, kBlock);
    const double hk = 0.5 * dt * kAcc / c->p.mass;
    if (phase == 0) {
        if (!d_pos_all) return fail(c, SC_ERR_INVALID, "sc_step_rows: d_pos_all is NULL%s");
        if (!c->have_vel || !c->forces_valid)
            return fail(c, SC_ERR_STATE, "sc_step_rows: phase 0 needs velocities and forces (phases 1, 2 with dt = 0 evaluate them)%s");
        kick_drift_kernel<<<nb_rows, kBlock, 0, c->stream>>>(c->xs, c->vel, c->force, c->scal, nullptr, c->xf, c->xfr, rb, re, hk, dt);
        export_rows_kernel<<<nb_rows, kBlock, 0, c->stream>>>(c->xs, d_pos_all, rb, re);
        SC_CUDA_CHECK(c, cudaGetLastError());
        c->launches += 2;
        c->density_valid = c->forces_valid = c->energy_valid = false;
        return SC_OK;
    }
    if (phase == 1) {
        if (!d_pos_all || !d_rho_all) return fail(c, SC_ERR_INVALID, "sc_step_rows: NULL all-atoms array%s");
        pack_positions_kernel<<<nb_all, kBlock, 0, c->stream>>>(d_pos_all, c->xs, c->xf, c->xfr, N);
        SC_CUDA_CHECK(c, cudaGetLastError());
        c->launches += 1;
        c->density_valid = c->forces_valid = c->energy_valid = false;
        sc_status st = run_sweep(c, false, false);
        if (st != SC_OK) return st;
        SC_CUDA_CHECK(c, cudaMemcpyAsync(d_rho_all + rb, c->rho + rb, sizeof(double) * size_t(rows), cudaMemcpyDeviceToDevice, c->stream));
        return SC_OK;
    }
    if (!d_rho_all) return fail(c, SC_ERR_INVALID, "sc_step_rows: d_rho_all is NULL%s");
    import_density_kernel<<<nb_all, kBlock, 0, c->stream>>>(d_rho_all, c->xs, c->xf, c->xfr, c->rho, N, c->consts.Bm);
    SC_CUDA_CHECK(c, cudaGetLastError());
    c->launches += 1;
    c->density_valid = true;
    if (c->emb_pending) {
        reduce_partials_kernel<<<1, 1024, 0, c->stream>>>(c->part_a, c->emb_pending, c->scal, kSlotEEmb, -c->consts.eps_c);
        SC_CUDA_CHECK(c, cudaGetLastError());
        c->launches += 1;
        c->emb_pending = 0;
    }
    sc_status st = run_sweep(c, true, true);
    if (st != SC_OK) return st;
    c->forces_valid = c->energy_valid = true;
    if (dt > 0.0) {
        if (!c->have_vel) return fail(c, SC_ERR_STATE, "sc_step_rows: velocities were never set%s");
        if (thermo == SC_THERMO_LANGEVIN) {
            LangevinArgs lg{};
            lg.c1 = std::exp(-th->gamma * dt);
            lg.c2 = std::sqrt((1.0 - lg.c1 * lg.c1) * kBoltzmann * th->T_end * kAcc / c->p.mass);
            lg.key0 = uint32_t(th->seed); lg.key1 = uint32_t(th->seed >> 32);
            lg.step_lo = uint32_t(c->langevin_step); lg.step_hi = uint32_t(c->langevin_step >> 32);
            lg.perm = nullptr;
            kick_langevin_ke_kernel<<<nb_rows, kBlock, 0, c->stream>>>(c->vel, c->force, c->part_ke, rb, re, hk, lg);
            c->langevin_step += 1;
        } else {
            kick_ke_kernel<<<nb_rows, kBlock, 0, c->stream>>>(c->vel, c->force, c->part_ke, rb, re, hk);
        }
        SC_CUDA_CHECK(c, cudaGetLastError());
        c->launches += 1;
    }
    return SC_OK;
}

sc_status sc_stats(sc_ctx *c, int64_t *n_rebuilds, int64_t *n_pairs_in_cut, int64_t *max_neighbours) {
    if (!c) return SC_ERR_INVALID;
    if (!c->cutoff) {
        if (n_rebuilds) *n_rebuilds = 0;
        if (n_pairs_in_cut) *n_pairs_in_cut = c->N * (c->N - 1);
        if (max_neighbours) *max_neighbours = c->N - 1;
        return SC_OK;
    }
    unsigned long long cnt[kNumCounters];
    SC_CUDA_CHECK(c, cudaMemcpyAsync(cnt, c->counters, sizeof(cnt), cudaMemcpyDeviceToHost, c->stream));
    SC_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    if (n_rebuilds) *n_rebuilds = int64_t(cnt[kCntRebuilds]);
    if (n_pairs_in_cut) *n_pairs_in_cut = int64_t(cnt[kCntPairsInCut]);
    if (max_neighbours) *max_neighbours = int64_t(cnt[kCntMaxRow]);
    if (cnt[kCntOverflow])
        return fail(c, SC_ERR_CAPACITY, "a neighbour row overflowed its capacity; results since then are invalid%s");
    return SC_OK;
}

sc_status sc_rdf(sc_ctx *c, const double *h_centre, double r_select, double bin_width, int32_t n_bins,
                 int64_t *h_counts, int64_t *h_n_ref, double *h_centre_used) {
    if (!c) return SC_ERR_INVALID;
    if (!c->have_pos) return fail(c, SC_ERR_STATE, "sc_rdf: no positions set%s");
    if (!h_counts || n_bins < 1 || n_bins > kRdfMaxBins || !(r_select > 0.0) || !(bin_width > 0.0) ||
        !std::isfinite(r_select) || !std::isfinite(bin_width))
        return fail(c, SC_ERR_INVALID, "sc_rdf: need h_counts, 1 <= n_bins <= 4096, r_select > 0, bin_width > 0%s");
    const int N = int(c->N);
    SC_CUDA_CHECK(c, cudaMemsetAsync(c->rdf_counts, 0, sizeof(unsigned long long) * (kRdfMaxBins + 2), c->stream));
    if (h_centre) {
        if (!std::isfinite(h_centre[0]) || !std::isfinite(h_centre[1]) || !std::isfinite(h_centre[2]))
            return fail(c, SC_ERR_INVALID, "sc_rdf: centre must be finite%s");
        SC_CUDA_CHECK(c, cudaMemcpyAsync(c->rdf_meta, h_centre, 3 * sizeof(double), cudaMemcpyHostToDevice, c->stream));
        SC_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));             // h_centre is pageable caller memory
    } else {
        rdf_centre_kernel<<<1, 1024, 0, c->stream>>>(c->xs, N, c->rdf_meta);
        c->launches += 1;
    }
    unsigned int *n_ref = reinterpret_cast<unsigned int *>(c->rdf_counts + kRdfMaxBins);
    rdf_select_kernel<<<ceil_div(N, kBlock), kBlock, 0, c->stream>>>(c->xs, N, c->rdf_meta, r_select * r_select, c->rdf_refs, n_ref);
    rdf_count_kernel<<<ceil_div(N, kRdfBlock), kRdfBlock, 0, c->stream>>>(c->xs, N, c->rdf_refs, n_ref, 1.0 / bin_width,
                                                                           int(n_bins), c->rdf_counts);
    SC_CUDA_CHECK(c, cudaGetLastError());
    c->launches += 2;
    std::vector<unsigned long long> host(size_t(n_bins) + 0);
    unsigned long long nref_word = 0;
    double centre[3];
    SC_CUDA_CHECK(c, cudaMemcpyAsync(host.data(), c->rdf_counts, sizeof(unsigned long long) * size_t(n_bins), cudaMemcpyDeviceToHost, c->stream));
    SC_CUDA_CHECK(c, cudaMemcpyAsync(&nref_word, c->rdf_counts + kRdfMaxBins, sizeof(unsigned long long), cudaMemcpyDeviceToHost, c->stream));
    SC_CUDA_CHECK(c, cudaMemcpyAsync(centre, c->rdf_meta, 3 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    SC_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    for (int b = 0; b < n_bins; ++b) h_counts[b] = int64_t(host[size_t(b)]);
    if (h_n_ref) *h_n_ref = int64_t(nref_word & 0xffffffffull);
    if (h_centre_used) { h_centre_used[0] = centre[0]; h_centre_used[1] = centre[1]; h_centre_used[2] = centre[2]; }
    return SC_OK;
}

sc_status sc_msd(sc_ctx *c, const double *d_ref_pos, double r_centre, int32_t align, double *h_msd, int64_t *h_n_sel,
                 double *h_rot) {
    if (!c) return SC_ERR_INVALID;
    if (!c->have_pos) return fail(c, SC_ERR_STATE, "sc_msd: no positions set%s");
    if (!d_ref_pos || !h_msd || align < 0 || align > 2 || std::isnan(r_centre))
        return fail(c, SC_ERR_INVALID, "sc_msd: need d_ref_pos, h_msd, align in 0..2, r_centre not NaN%s");
    const int N = int(c->N);
    const int nb = int(std::min<int64_t>(ceil_div(c->N, kMsdBlock), kMsdMaxBlocks));
    const int *perm = c->cutoff ? c->perm : nullptr;
    double *p0 = c->msd_part, *p1 = p0 + size_t(kMsdMaxBlocks) * kMsdPartStride, *p2 = p1 + size_t(kMsdMaxBlocks) * kMsdPartStride;
    const double rc2 = r_centre > 0.0 ? r_centre * r_centre : 0.0;
    msd_centroid_kernel<<<nb, kMsdBlock, 0, c->stream>>>(c->xs, d_ref_pos, perm, N, p0);
    msd_covariance_kernel<<<nb, kMsdBlock, 0, c->stream>>>(c->xs, d_ref_pos, perm, N, int(align), p0, p1, c->msd_meta);
    msd_rotation_kernel<<<1, 32, 0, c->stream>>>(p1, nb, int(align), c->msd_meta);
    msd_accumulate_kernel<<<nb, kMsdBlock, 0, c->stream>>>(c->xs, d_ref_pos, perm, N, rc2, c->msd_meta, p2);
    msd_total_kernel<<<1, 32, 0, c->stream>>>(p2, nb, c->msd_meta);
    SC_CUDA_CHECK(c, cudaGetLastError());
    c->launches += 5;
    double meta[17];
    SC_CUDA_CHECK(c, cudaMemcpyAsync(meta, c->msd_meta, sizeof(meta), cudaMemcpyDeviceToHost, c->stream));
    SC_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    const double cnt = meta[16];
    *h_msd = cnt > 0.0 ? meta[15] / cnt : 0.0;
    if (h_n_sel) *h_n_sel = int64_t(cnt);
    if (h_rot) for (int q = 0; q < 9; ++q) h_rot[q] = meta[6 + q];
    if (!std::isfinite(meta[15])) return fail(c, SC_ERR_NONFINITE, "sc_msd: the displacement sum is not finite%s");
    return SC_OK;
}

sc_status sc_eval_host(sc_ctx *c, const double *h_pos, double *h_force, double *h_rho, double *h_epot) {
    if (!c || !h_pos) return fail(c, SC_ERR_INVALID, "sc_eval_host: h_pos is NULL%s");
    const size_t n = size_t(c->N);
    SC_CUDA_CHECK(c, cudaMemcpyAsync(c->stage_a, h_pos, sizeof(double) * 3 * n, cudaMemcpyHostToDevice, c->stream));
    sc_status st = sc_set_state(c, c->stage_a, nullptr);
    if (st != SC_OK) return st;
    st = ensure_forces(c, true);
    if (st != SC_OK) return st;
    const double *src_f = c->force, *src_r = c->rho;
    if (c->cutoff) {                      // back to the caller's order through the staging buffers
        if (h_force) { st = copy_out(c, c->force, c->stage_b, 3); if (st != SC_OK) return st; src_f = c->stage_b; }
        if (h_rho) { st = copy_out(c, c->rho, c->stage_a, 1); if (st != SC_OK) return st; src_r = c->stage_a; }
    }
    if (h_force) SC_CUDA_CHECK(c, cudaMemcpyAsync(h_force, src_f, sizeof(double) * 3 * n, cudaMemcpyDeviceToHost, c->stream));
    if (h_rho) SC_CUDA_CHECK(c, cudaMemcpyAsync(h_rho, src_r, sizeof(double) * n, cudaMemcpyDeviceToHost, c->stream));
    double s[2];
    st = read_scalars(c, s, 2);
    if (st != SC_OK) return st;
    if (h_epot) *h_epot = s[kSlotEPair] + s[kSlotEEmb];
    if (!std::isfinite(s[0] + s[1])) return fail(c, SC_ERR_NONFINITE, "sc_eval_host: potential energy is not finite%s");
    return check_flags(c);
}

sc_status sc_step_host(sc_ctx *c, double *h_pos, double *h_vel, double dt_fs, const sc_thermostat *thermostat,
                       int64_t nsteps, double *h_scalars) {
    if (!c || !h_pos || !h_vel) return fail(c, SC_ERR_INVALID, "sc_step_host: NULL state pointer%s");
    const size_t n = size_t(c->N);
    SC_CUDA_CHECK(c, cudaMemcpyAsync(c->stage_a, h_pos, sizeof(double) * 3 * n, cudaMemcpyHostToDevice, c->stream));
    SC_CUDA_CHECK(c, cudaMemcpyAsync(c->stage_b, h_vel, sizeof(double) * 3 * n, cudaMemcpyHostToDevice, c->stream));
    sc_status st = sc_set_state(c, c->stage_a, c->stage_b);
    if (st != SC_OK) return st;
    st = do_step(c, dt_fs, thermostat, nsteps);
    if (st != SC_OK) return st;
    st = ensure_forces(c, true);
    if (st != SC_OK) return st;
    st = sc_get_state(c, c->stage_a, nullptr);
    if (st != SC_OK) return st;
    SC_CUDA_CHECK(c, cudaMemcpyAsync(h_pos, c->stage_a, sizeof(double) * 3 * n, cudaMemcpyDeviceToHost, c->stream));
    st = copy_out(c, c->vel, c->stage_b, 3);
    if (st != SC_OK) return st;
    SC_CUDA_CHECK(c, cudaMemcpyAsync(h_vel, c->stage_b, sizeof(double) * 3 * n, cudaMemcpyDeviceToHost, c->stream));
    if (h_scalars) {
        double ke = 0, temp = 0;
        st = sc_kinetic(c, &ke, &temp);
        if (st != SC_OK) return st;
        double s[2];
        st = read_scalars(c, s, 2);
        if (st != SC_OK) return st;
        h_scalars[0] = s[0] + s[1]; h_scalars[1] = ke; h_scalars[2] = temp;
        if (!std::isfinite(h_scalars[0])) return fail(c, SC_ERR_NONFINITE, "sc_step_host: potential energy is not finite%s");
    } else {
        SC_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    }
    return SC_OK;
}

sc_status sc_launch_count(sc_ctx *c, int64_t *n_launches) {
    if (!c || !n_launches) return SC_ERR_INVALID;
    *n_launches = c->launches;
    return SC_OK;
}

sc_status sc_profile(sc_ctx *c, int32_t enable) {
    if (!c) return SC_ERR_INVALID;
    c->profile = enable != 0;
    return SC_OK;
}

sc_status sc_profile_read(sc_ctx *c, double *h_ms_density, double *h_ms_force) {
    if (!c) return SC_ERR_INVALID;
    SC_CUDA_CHECK(c, cudaStreamSynchronize(c->stream));
    float a = 0.f, b = 0.f;
    if (cudaEventElapsedTime(&a, c->ev[0], c->ev[1]) != cudaSuccess ||
        cudaEventElapsedTime(&b, c->ev[1], c->ev[2]) != cudaSuccess)
        return fail(c, SC_ERR_STATE, "sc_profile_read: no profiled sweep recorded%s");
    if (h_ms_density) *h_ms_density = a;
    if (h_ms_force) *h_ms_force = b;
    return SC_OK;
}

}  // extern "C"
