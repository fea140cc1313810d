// lrmd.cu — the C ABI of include/lrmd.h: argument validation, workspace layout, integrator
// substage sequencing (eq.(4) and the 12-step listing) and kernel launches.
// All arithmetic of the method runs in the kernels of hmf_kernels.cuh / pair_kernels.cuh; the
// host only computes the four products B*dt, D*dt per call and chooses launch shapes.
#include "../../include/lrmd.h"

#include <cmath>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <tuple>
#include <utility>
#include <vector>

#include "hmf_kernels.cuh"
#include "pair_kernels.cuh"
#include "band_kernels.cuh"
#include "peak_kernels.cuh"

namespace {

using namespace lrmd;

constexpr int kNumSm = 148;                 // B200
constexpr size_t kAlign = 256;
constexpr int kEnergyGrid = kNumSm * 4;     // CTAs of the kinetic-energy partial kernel
constexpr int kGraphSteps = 8;              // steady-state steps per replayed CUDA graph
constexpr size_t kMaxTimedEvents = 1 << 15; // LRMD_OPT_KERNEL_TIMING: at most 16384 timed launches between reads

inline size_t align_up(size_t x) { return (x + kAlign - 1) / kAlign * kAlign; }

struct Layout {
    size_t hmf_partial = 0;   // 3 rotating buffers of kHmfMaxGrid double2 (HMF)
    size_t js = 0;            // packed j-stream double2[N] (pair models)
    size_t js32 = 0;          // fp32 copy float2[N + pad] (GRAV2D, pair precision 1)
    size_t partial0 = 0;      // [slots][N] partial forces
    size_t partial1 = 0;      // [slots][N] (GRAV2D)
    size_t kpart = 0;         // 3 * kEnergyGrid
    size_t vpart = 0;         // one per CTA of the pair-energy kernel
    size_t shared2 = 0;       // HMF shard: this rank's (sum cos, sum sin), all-reduced in place
    size_t sym_wstart = 0, sym_tiles = 0, ipart0 = 0, ipart1 = 0, jpart0 = 0, jpart1 = 0;   // symmetric kernel
    size_t band_wpiece = 0, band_pieces = 0, band_infos = 0, bibuf0 = 0, bibuf1 = 0, bjbuf0 = 0, bjbuf1 = 0;   // band kernel
    size_t total = 0;
};

}  // namespace

struct lrmd_ctx {
    int model = 0;
    int64_t N = 0;              // particles this context owns (all of them unless it is a shard)
    double eps = 0.0;
    // sharding (lrmd_set_shard): this context owns the global indices i0 .. i0 + N - 1 of N_total particles
    int64_t N_total = 0, i0 = 0;
    lrmd_allreduce_fn allreduce = nullptr;
    lrmd_allgather_fn allgather = nullptr;
    void* coll_user = nullptr;
    // options as set (0 / -1 = choose)
    int64_t opt_precision = 0, opt_pair_ctas = 0, opt_graph = -1, opt_hmf_grid = 0;
    int64_t opt_hmf_variant = -1, opt_pair_variant = -1, opt_sym = -1, opt_sym_tiles = 0, opt_fuse = -1, opt_sym_xch = -1;
    int64_t opt_band_height = 0;
    // resolved
    int hmf_grid = 0, hmf_variant = 0, pair_variant = 0;
    int slots = 1;              // partial force rows per particle (pair models)
    lrmd::PairPart part{};      // work partition of the pair kernels
    bool sym = false;           // symmetric (Newton's third law) force kernel in use
    lrmd::SymPart spart{};      // its work partition; the two tables below are uploaded by lrmd_set_workspace
    std::vector<int4> sym_wstart;
    std::vector<int2> sym_tiles;
    std::vector<int4> sym_batches;   // (first tile, end tile, first worker, workers) per launch
    int sym_slots = 1, sym_R = 4, sym_rows = 1;
    int sym_xch = 3;            // LRMD_OPT_PAIR_SYM_EXCHANGE as resolved
    bool band = false;          // band kernel (band_kernels.cuh) in use for the force; the tables below are uploaded
    lrmd::BandPart bpart{};     //   by lrmd_set_workspace
    std::vector<int> band_wpiece;
    std::vector<lrmd::BandPiece> band_pieces;
    std::vector<lrmd::BandInfo> band_infos;
    std::vector<int> band_owner;     // worker of every piece (diagnostics)
    int band_R = 8;
    size_t band_jrow = 0;       // elements of all bands' j-side rows
    bool use_graph = false;
    bool grid_unavailable = false;   // a cooperative launch of the grid-resident HMF kernel failed: not tried again
    Layout lay;
    // bindings
    char* ws = nullptr;
    double *a0 = nullptr, *a1 = nullptr, *a2 = nullptr, *a3 = nullptr;
    bool state_set = false;
    bool force_valid = false;   // HMF: hmf_partial[cur] holds the sums at theta; pair: partial* hold F(q)
    bool js_valid = false;      // pair models: js[] matches q
    bool v_valid = false;       // band kernel: vpart[0 .. P) holds the potential at q (the last force evaluation delivered it)
    bool want_v = false;        // lrmd_step_observe: the force evaluation that ends lrmd_step delivers V as well
    int cur = 0;                // HMF: which of the 3 partial buffers is current
    // cached CUDA graph of kGraphSteps steady-state steps (HMF)
    cudaGraphExec_t graph_exec = nullptr;
    double graph_dt = 0.0;
    int graph_cur = -1;
    int64_t graph_nodes = 0;
    // bookkeeping
    int64_t launches = 0;
    int cuda_err = 0;
    std::vector<const void*> smem_ready;   // kernels whose dynamic shared-memory limit has been raised
    // LRMD_OPT_KERNEL_TIMING: event pairs around the dominant kernel's launches
    bool timing = false;
    std::vector<cudaEvent_t> ev;      // 2 per timed launch (start, stop), created on demand
    size_t ev_used = 0;
};

namespace {

// ---- option resolution -------------------------------------------------------------------------------

// Launch shapes compiled in (chosen from LRMD_OPT_HMF_VARIANT / LRMD_OPT_PAIR_VARIANT / LRMD_OPT_PAIR_CTAS sweeps on B200;
// the options stay settable so that the choice can be re-measured with bench.py).
// HMF: variant 0 is the register-prefetch kernel, 1-2 the TMA-staged kernel <consumer threads, stages, CTAs per
// SM> (N >= 1e6), 3 the cluster-resident kernel (N <= 20,480: the step is latency-bound).
struct HmfVariant { int consumers, stages, minb; };
constexpr HmfVariant kHmfVariants[] = {{0, 0, 0}, {512, 4, 1}, {256, 6, 2}, {-1, 0, 0}, {-2, 0, 0}};
constexpr int kHmfClusterVariant = 3;   // cluster-resident kernel: whole state in registers, all steps in one launch
constexpr int kHmfGridVariant = 4;      // grid-resident kernel: whole state in shared memory, one cooperative launch per call
constexpr int64_t kHmfGridMaxN = (int64_t)kNumSm * kHmfGridMaxLocal;   // 1,070,336
constexpr int64_t kHmfClusterMaxN = (int64_t)kHmfClusterCtas * kHmfClusterThreads * 8;   // 20,480
constexpr int kNumHmfVariants = sizeof(kHmfVariants) / sizeof(kHmfVariants[0]);
constexpr int64_t kHmfTmaMinN = 1000000;
constexpr double kSymRowBytes = 1073741824.0;   // scratch for the symmetric kernel's j-side rows per launch (1 GiB)

// Pair kernels: <threads, i per thread, j per stage, CTAs per SM, j unroll>.
using PairCfg0 = PairCfg<128, 4, 256, 4, 4>;   // Ring default (88 registers)
using PairCfg1 = PairCfg<128, 8, 256, 2, 2>;   // 2D default: one LDS.128 per 8 pairs
using PairCfg2 = PairCfg<256, 4, 256, 2, 4>;
constexpr int kNumPairVariants = 3;

template <typename F>
void with_pair_cfg(int v, F f) {
    switch (v) {
        case 1: f(PairCfg1{}); break;
        case 2: f(PairCfg2{}); break;
        default: f(PairCfg0{}); break;
    }
}

// Symmetric force kernel (row N4): decide whether it is used and build its work tables.
// Units are (tile, chunk) pairs in tile-major order, chunk >= tile * R; G workers get equal contiguous shares.
void resolve_sym(lrmd_ctx* c, bool rows_needed) {
    // rows_needed = false: the band kernel evaluates the force; the tables built here then serve the symmetric
    // potential-energy kernel only (one launch, no partial force rows)
    c->sym = false;
    c->sym_wstart.clear();
    c->sym_tiles.clear();
    c->sym_batches.clear();
    const int64_t N = c->N;
    if (c->opt_sym == 0 || c->N_total != c->N) return;
    if (c->model == LRMD_RING && c->opt_precision == 1) return;    // Ring, fp32 pairs: ordered kernel only
    if (c->opt_sym < 0 && N < 2048) return;    // small systems: the ordered kernel's one wave is as fast
    // i per lane: Ring 4, 2D 8 (measured best of the two); launch shape 0 / 1 asks for 4 / 8
    const int R = c->opt_pair_variant == 0 ? 4 : (c->opt_pair_variant == 1 ? 8 : (c->model == LRMD_RING ? 4 : 8));
    const int T = 32 * R;
    const int64_t ntiles = (N + T - 1) / T, nchunks = (N + 31) / 32;
    const int comps = c->model == LRMD_GRAV2D ? 2 : 1;
    // The j-side rows cost N doubles per component and tile.  Tiles are processed in batches of TB tiles (one
    // kernel launch + one fold per batch) so that the rows of a batch fit kSymRowBytes: one batch up to
    // N ~ 1.8e5 (2D), 64 batches at N = 2^20.
    int64_t TB = (int64_t)(kSymRowBytes / ((double)N * 8.0 * comps));
    if (c->opt_sym_tiles > 0) TB = c->opt_sym_tiles;
    if (!rows_needed) TB = ntiles;
    if (TB < 1) TB = 1;
    if (TB > ntiles) TB = ntiles;
    // workers per launch: 32 per SM (4 waves of the 8 resident warps); at least two units each
    int64_t Gwant = c->opt_pair_ctas > 0 ? c->opt_pair_ctas : (int64_t)kNumSm * 32;
    // the host-built work table has one entry per worker and launch: keep it below 2^22 entries (64 MB)
    const int64_t nbatches = (ntiles + TB - 1) / TB;
    if (!rows_needed) Gwant = (int64_t)kNumSm * 32;
    if (c->opt_pair_ctas <= 0 && rows_needed) {
        // a tile's i-side rows number about workers / tiles per launch: keep them within ~4 GiB
        int64_t maxslots = (int64_t)(4.0 * 1073741824.0 / ((double)N * 8.0 * comps));
        if (maxslots < 8) maxslots = 8;
        if (Gwant > maxslots * TB) Gwant = maxslots * TB;
        if (Gwant < (int64_t)kNumSm * 8) Gwant = (int64_t)kNumSm * 8;
    }
    if (c->opt_pair_ctas <= 0 && nbatches * Gwant > ((int64_t)1 << 22)) {
        Gwant = ((int64_t)1 << 22) / nbatches;
        if (Gwant < (int64_t)kNumSm * 8) return;    // launches would not fill the GPU (N beyond ~8e6): ordered kernel
    }
    if (nbatches * Gwant > ((int64_t)1 << 26)) return;
    c->sym_tiles.assign((size_t)ntiles, make_int2(0x7fffffff, -1));
    int gmax = 1;
    for (int64_t t0 = 0; t0 < ntiles; t0 += TB) {
        const int64_t t1 = t0 + TB < ntiles ? t0 + TB : ntiles;
        int64_t U = 0;
        for (int64_t a = t0; a < t1; ++a) U += nchunks - a * R;
        int64_t G = Gwant;
        if ((c->opt_pair_ctas <= 0 || !rows_needed) && G > U / 2) G = U / 2;
        if (G > U) G = U;
        if (G < 1) G = 1;
        const int64_t w0 = (int64_t)c->sym_wstart.size();
        c->sym_batches.push_back(make_int4((int)t0, (int)t1, (int)w0, (int)G));
        if (G > gmax) gmax = (int)G;
        int64_t a = t0, cum = 0;     // cum = units of the batch before tile a
        for (int64_t w = 0; w < G; ++w) {
            const int64_t u0 = (w * U) / G, u1 = ((w + 1) * U) / G;
            while (u0 >= cum + (nchunks - a * R)) { cum += nchunks - a * R; ++a; }
            c->sym_wstart.push_back(make_int4((int)a, (int)(a * R + (u0 - cum)), (int)(u1 - u0), 0));
            const int gw = (int)(w0 + w);     // global worker index: slots are counted from a tile's first worker
            int64_t aa = a, cc = cum;
            for (;;) {
                int2& r = c->sym_tiles[(size_t)aa];
                if (gw < r.x) r.x = gw;
                if (gw > r.y) r.y = gw;
                if (u1 <= cc + (nchunks - aa * R)) break;
                cc += nchunks - aa * R;
                ++aa;
            }
        }
    }
    int smax = 1;
    for (const int2& r : c->sym_tiles) if (r.y - r.x + 1 > smax) smax = r.y - r.x + 1;
    c->sym_slots = smax;
    c->sym_xch = c->opt_sym_xch >= 0 ? (int)c->opt_sym_xch : 3;
    c->sym_R = R;
    c->sym_rows = (int)TB;
    lrmd::SymPart S;
    S.N = N; S.T = T; S.ntiles = (int)ntiles; S.nchunks = (int)nchunks; S.G = gmax; S.w0 = 0; S.tile0 = 0; S.tile1 = (int)ntiles;
    S.wstart = nullptr; S.tile_rng = nullptr;
    c->spart = S;
    c->sym = true;
}

// Band kernel (band_kernels.cuh): choose the band height, cut every band's columns into pieces of equal weight and
// assign them to the P workers in band-major order.  Weight of one 32-column chunk in column block blk of band A:
// 11 (2D) or 12 (Ring) FP64 instructions per pair for every I-block of the band above the block, 9 / 11 for the block
// itself if it is in the band (DIAG walk: every ordered pair, i-side only).
constexpr int64_t kBandMinN = 49152;     // default: band kernel from this N on (unsharded fp64 contexts)
constexpr double kBandL2Bytes = 80.0 * 1048576.0;   // i-side rows all CTAs cycle through: kept within L2

void resolve_band(lrmd_ctx* c) {
    c->band = false;
    c->band_wpiece.clear();
    c->band_pieces.clear();
    c->band_infos.clear();
    c->band_owner.clear();
    const int64_t N = c->N;
    if (c->opt_sym == 0 || c->opt_sym == 1 || c->N_total != c->N) return;
    if (c->opt_precision != 0 && c->model != LRMD_GRAV2D) return;     // fp32 pairs: the band kernel exists for 2D only
    if (c->opt_sym < 0 && N < kBandMinN) return;
    // rows per lane: 8 for both models (Ring measured 7.7 % faster than with 4 at N = 512,000); launch shape 0 asks for 4
    int R = c->opt_pair_variant == 0 ? 4 : 8;
    if (c->opt_precision == 1 && c->opt_pair_variant == 2) R = 16;      // fp32 pairs: experimental 16 rows per lane
    const int64_t IB = (int64_t)kBandWarps * 32 * R, JB = IB / 32;
    const int64_t nIB = (N + IB - 1) / IB, nchunks = (N + 31) / 32;
    if (nIB > (1 << 20)) return;
    const int64_t P = c->opt_pair_ctas > 0 ? c->opt_pair_ctas : (R == 16 ? 1 : 2) * (int64_t)kNumSm;
    // band height: the i-side rows cost (pieces ~ P + bands) x hb x IB elements, the j-side rows ~ bands x N / 2.  A CTA
    // adds to its piece's i-side row once per (J-block, I-block) visit, cycling through hb x IB rows: the height is
    // capped so that the rows all CTAs cycle through stay in L2 (kBandL2Bytes of the 126 MB), else every visit would
    // take 64 KB through HBM (8.5 GB per force evaluation at N = 2^20 with the unconstrained height 21; ncu, profiles/).
    const int comps = c->model == LRMD_GRAV2D ? 2 : 1;
    int64_t hb = 1;
    if (c->opt_band_height > 0) {
        hb = c->opt_band_height < nIB ? c->opt_band_height : nIB;
    } else {
        int64_t hmax = (int64_t)(kBandL2Bytes / ((double)P * (double)IB * 8.0 * comps));
        if (hmax < 1) hmax = 1;
        auto elements = [&](int64_t h) {
            const double nb = (double)((nIB + h - 1) / h);
            return ((double)P + nb) * (double)h * (double)IB + nb * 0.5 * (double)N;
        };
        double best = -1.0, best_l2 = -1.0;
        int64_t h_l2 = 1;
        for (int64_t h = 1; h <= nIB; ++h) {
            const double cost = elements(h);
            if (best < 0.0 || cost < best) { best = cost; hb = h; }
            if (h <= hmax && (best_l2 < 0.0 || cost < best_l2)) { best_l2 = cost; h_l2 = h; }
        }
        // beyond ~1 GiB of rows the L2-resident height costs more memory than the HBM round trips are worth
        // (64 KB per 4.2e6 pair evaluations)
        if (best_l2 * 8.0 * comps <= 1073741824.0) hb = h_l2;
    }
    const int64_t nbands = (nIB + hb - 1) / hb;
    const int64_t wsym = c->model == LRMD_RING ? 12 : 11, wdiag = c->model == LRMD_RING ? 11 : 9;
    auto chunk_weight = [&](int64_t blk0, int64_t nblk, int64_t blk) {
        int64_t nsym = blk - blk0 < nblk ? blk - blk0 : nblk;
        return wsym * nsym + (blk < blk0 + nblk ? wdiag : 0);
    };
    double wtot = 0.0;      // exact in double: below 2^53 for every N the pair models accept
    for (int64_t A = 0; A < nbands; ++A) {
        const int64_t blk0 = A * hb, nblk = blk0 + hb <= nIB ? hb : nIB - blk0;
        for (int64_t blk = blk0; blk < nIB; ++blk) {
            const int64_t cb = blk * JB, ce = (blk + 1) * JB < nchunks ? (blk + 1) * JB : nchunks;
            wtot += (double)(chunk_weight(blk0, nblk, blk) * (ce - cb));
        }
    }
    c->band_wpiece.assign((size_t)P + 1, 0);
    int64_t w = 0;
    double cum = 0.0;
    auto boundary = [&](int64_t k) { return std::floor(wtot * (double)k / (double)P); };
    double next = boundary(1);
    size_t jrow = 0;
    for (int64_t A = 0; A < nbands; ++A) {
        const int64_t blk0 = A * hb, nblk = blk0 + hb <= nIB ? hb : nIB - blk0;
        BandInfo info;
        info.blk0 = (int)blk0; info.nblk = (int)nblk; info.pf0 = (int)c->band_pieces.size(); info.pf1 = 0;
        info.cstart = (int)(blk0 * JB); info.pad = 0;
        info.joff = (long long)jrow;
        jrow += (size_t)((nchunks - blk0 * JB) * 32 + 31) / 32 * 32;
        int64_t start = blk0 * JB;
        auto close_piece = [&](int64_t end) {
            if (end > start) {
                BandPiece pc;
                pc.band = (int)A; pc.c0 = (int)start; pc.c1 = (int)end; pc.pad = 0;
                c->band_pieces.push_back(pc);
                c->band_owner.push_back((int)w);
                start = end;
            }
        };
        for (int64_t blk = blk0; blk < nIB; ++blk) {
            const int64_t ce = (blk + 1) * JB < nchunks ? (blk + 1) * JB : nchunks;
            const double wt = (double)chunk_weight(blk0, nblk, blk);
            int64_t cpos = blk * JB;
            while (cpos < ce) {
                int64_t take = ce - cpos;
                if (w < P - 1) {
                    const int64_t need = (int64_t)std::ceil((next - cum) / wt);     // chunks up to the worker's boundary
                    if (need < take) take = need < 1 ? 1 : need;
                }
                cum += wt * (double)take;
                cpos += take;
                while (w < P - 1 && cum >= next) {       // the worker's share is complete: the next one starts here
                    close_piece(cpos);
                    ++w;
                    c->band_wpiece[(size_t)w] = (int)c->band_pieces.size();
                    next = boundary(w + 1);
                }
            }
        }
        close_piece(nchunks);
        info.pf1 = (int)c->band_pieces.size();
        c->band_infos.push_back(info);
    }
    for (int64_t k = w + 1; k <= P; ++k) c->band_wpiece[(size_t)k] = (int)c->band_pieces.size();
    lrmd::BandPart B;
    B.N = N; B.istride = hb * IB; B.IB = (int)IB; B.nIB = (int)nIB; B.nchunks = (int)nchunks; B.nbands = (int)nbands;
    B.hb = (int)hb; B.P = (int)P; B.wpiece = nullptr; B.pieces = nullptr; B.bands = nullptr;
    c->bpart = B;
    c->band_R = R;
    c->band_jrow = jrow;
    c->band = true;
}

void resolve(lrmd_ctx* c) {
    const int64_t N = c->N;
    Layout L;
    size_t off = 0;
    if (c->model == LRMD_HMF) {
        const bool sharded = c->N_total != c->N;
        c->hmf_variant = c->opt_hmf_variant >= 0 ? (int)c->opt_hmf_variant
                         : (N <= kHmfClusterMaxN ? kHmfClusterVariant
                            : ((N <= kHmfGridMaxN && !sharded && !c->grid_unavailable) ? kHmfGridVariant
                               : (N >= kHmfTmaMinN ? 1 : 0)));
        if (c->hmf_variant == kHmfClusterVariant && (N > kHmfClusterMaxN || sharded)) c->hmf_variant = 0;
        if (c->hmf_variant == kHmfGridVariant && (N > kHmfGridMaxN || sharded || c->grid_unavailable))
            c->hmf_variant = N >= kHmfTmaMinN ? 1 : 0;
        const HmfVariant hv = kHmfVariants[c->hmf_variant];
        int64_t g;
        if (c->hmf_variant == kHmfGridVariant) {
            g = kNumSm;        // one CTA per SM; the other HMF kernels read this many partials
        } else if (c->hmf_variant == kHmfClusterVariant) {
            // the other HMF kernels of this context (forces, energy) read this many partials
            g = c->opt_hmf_grid == kHmfClusterCtasMax ? kHmfClusterCtasMax : kHmfClusterCtas;
        } else if (c->hmf_variant == 0) {
            const int64_t nvec = N >> 2;
            g = c->opt_hmf_grid > 0 ? c->opt_hmf_grid : (nvec + kHmfThreads - 1) / kHmfThreads;
        } else {
            const int64_t chunk = 4 * (int64_t)hv.consumers;
            const int64_t nchunks = ((N & ~(int64_t)1) + chunk - 1) / chunk;
            g = c->opt_hmf_grid > 0 ? c->opt_hmf_grid : (int64_t)kNumSm * hv.minb;
            if (g > nchunks) g = nchunks;
        }
        if (g < 1) g = 1;
        if (g > kHmfMaxGrid) g = kHmfMaxGrid;
        c->hmf_grid = (int)g;
        c->slots = 1;
        L.hmf_partial = off; off = align_up(off + 3 * sizeof(double2) * kHmfMaxGrid);
        // replaying a captured graph of 8 steps removes the launch gaps between substages: 4 % at N = 1e7, 1 % at 5e7
        c->use_graph = c->opt_graph < 0 ? true : (c->opt_graph != 0);
        if (c->hmf_variant == kHmfClusterVariant || c->hmf_variant == kHmfGridVariant || sharded) c->use_graph = false;   // (collectives between substages)
        L.shared2 = off; off = align_up(off + sizeof(double2));
    } else {
        c->pair_variant = c->opt_pair_variant >= 0 ? (int)c->opt_pair_variant : (c->model == LRMD_GRAV2D ? 1 : 0);
        int itile = 0, minb = 0;
        with_pair_cfg(c->pair_variant, [&](auto cfg) { itile = decltype(cfg)::ITILE; minb = decltype(cfg)::MINB; });
        const int64_t itiles = (N + itile - 1) / itile;
        const int64_t NJ = c->N_total;                         // j runs over all particles, also in a shard
        const int64_t Lpos = itiles * NJ;                      // flattened (i-tile, j) positions
        const int64_t slots_hw = (int64_t)kNumSm * minb;       // resident CTAs on the device
        int64_t G;
        if (c->opt_pair_ctas > 0) {
            G = c->opt_pair_ctas;
        } else {
            // one wave of equal ranges for small N; for large N ranges of about max(64Ki, N/8) positions
            // (whole waves), which bounds both the tail of the last wave and the partial rows per tile
            int64_t qt = NJ / 8 > 65536 ? NJ / 8 : 65536;
            int64_t waves = (Lpos + slots_hw * qt / 2) / (slots_hw * qt);
            if (waves < 1) waves = 1;
            G = slots_hw * waves;
            const int64_t gmax = Lpos / 64 > 1 ? Lpos / 64 : 1;   // at least 64 j per CTA
            if (G > gmax) G = gmax;
        }
        if (G > Lpos) G = Lpos;
        if (G < 1) G = 1;
        PairPart P;
        P.N = NJ; P.Ni = N; P.i0 = c->i0; P.G = (int)G; P.q = Lpos / G; P.r = Lpos % G; P.itile = itile;
        c->part = P;
        int64_t smax = 1;
        for (int64_t t = 0; t < itiles; ++t) {
            long long first, last;
            part_tile_ctas(P, t, first, last);
            if (last - first + 1 > smax) smax = last - first + 1;
        }
        c->slots = (int)smax;
        c->hmf_grid = 0;
        (void)minb;
        resolve_band(c);
        resolve_sym(c, !c->band);
        L.js = off; off = align_up(off + sizeof(double2) * (size_t)NJ);
        if (c->opt_precision == 1) { L.js32 = off; off = align_up(off + sizeof(float2) * ((size_t)NJ + 2)); }
        const bool two = c->model == LRMD_GRAV2D;
        const size_t rows = c->sym ? 1 : (size_t)c->slots;     // symmetric: one folded row
        L.partial0 = off; off = align_up(off + sizeof(double) * (size_t)N * rows);
        if (two) { L.partial1 = off; off = align_up(off + sizeof(double) * (size_t)N * rows); }
        if (c->band) {
            L.band_wpiece = off; off = align_up(off + sizeof(int) * c->band_wpiece.size());
            L.band_pieces = off; off = align_up(off + sizeof(BandPiece) * c->band_pieces.size());
            L.band_infos = off; off = align_up(off + sizeof(BandInfo) * c->band_infos.size());
            const size_t irow = c->band_pieces.size() * (size_t)c->bpart.istride;
            L.bibuf0 = off; off = align_up(off + sizeof(double) * irow);
            if (two) { L.bibuf1 = off; off = align_up(off + sizeof(double) * irow); }
            L.bjbuf0 = off; off = align_up(off + sizeof(double) * c->band_jrow);
            if (two) { L.bjbuf1 = off; off = align_up(off + sizeof(double) * c->band_jrow); }
        }
        if (c->sym) {
            L.sym_wstart = off; off = align_up(off + sizeof(int4) * c->sym_wstart.size());
            L.sym_tiles = off; off = align_up(off + sizeof(int2) * c->sym_tiles.size());
        }
        if (c->sym && !c->band) {
            L.ipart0 = off; off = align_up(off + sizeof(double) * (size_t)N * c->sym_slots);
            if (two) { L.ipart1 = off; off = align_up(off + sizeof(double) * (size_t)N * c->sym_slots); }
            L.jpart0 = off; off = align_up(off + sizeof(double) * (size_t)N * c->sym_rows);
            if (two) { L.jpart1 = off; off = align_up(off + sizeof(double) * (size_t)N * c->sym_rows); }
        }
        size_t nv = (size_t)G;
        if (c->sym && c->sym_wstart.size() > nv) nv = c->sym_wstart.size();
        if (c->band && (size_t)c->bpart.P > nv) nv = (size_t)c->bpart.P;
        L.vpart = off; off = align_up(off + sizeof(double) * nv);
        c->use_graph = false;
    }
    L.kpart = off; off = align_up(off + sizeof(double) * 3 * kEnergyGrid);
    L.total = off;
    c->lay = L;
}

// After resolve(): the bound workspace stays valid only if every offset is unchanged and no device-resident work table
// (symmetric kernel) was rebuilt; otherwise the context returns to "workspace not set" (lrmd.h, lrmd_set_workspace).
void rebind_if_changed(lrmd_ctx* c, const Layout& before, bool had_sym) {
    // (a context that uses the band kernel also has c->sym set: the symmetric energy kernel's tables)
    if (std::memcmp(&before, &c->lay, sizeof(Layout)) != 0 || had_sym || c->sym) c->ws = nullptr;
}

void drop_graph(lrmd_ctx* c) {
    if (c->graph_exec) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }
    c->graph_cur = -1;
    c->graph_nodes = 0;
}

// ---- launcher: the same call either enqueues on a stream or appends a kernel node to a graph ---------

struct Launcher {
    lrmd_ctx* c;
    cudaStream_t stream;
    cudaGraph_t graph = nullptr;       // non-null: build mode
    cudaGraphNode_t last = nullptr;
    int64_t nodes = 0;
    int rc = LRMD_OK;

    size_t smem = 0;                   // dynamic shared memory of the next launch (reset after it)

    template <typename... KA, typename... A>
    void go(void (*kernel)(KA...), dim3 grid, dim3 block, A... a) {
        static_assert(sizeof...(KA) == sizeof...(A), "argument count");
        const size_t shmem = smem;
        smem = 0;
        if (rc != LRMD_OK) return;
        if (shmem > 48 * 1024) {
            bool ready = false;
            for (const void* k : c->smem_ready) ready = ready || k == (const void*)kernel;
            if (!ready) {
                const cudaError_t ea = cudaFuncSetAttribute((const void*)kernel,
                                                            cudaFuncAttributeMaxDynamicSharedMemorySize, (int)shmem);
                if (ea != cudaSuccess) { c->cuda_err = (int)ea; rc = LRMD_ECUDA; (void)cudaGetLastError(); return; }
                c->smem_ready.push_back((const void*)kernel);
            }
        }
        std::tuple<KA...> vals{static_cast<KA>(a)...};
        void* ptrs[sizeof...(KA)];
        fill(ptrs, vals, std::index_sequence_for<KA...>{});
        cudaError_t e;
        if (graph) {
            cudaKernelNodeParams kp;
            std::memset(&kp, 0, sizeof(kp));
            kp.func = (void*)kernel;
            kp.gridDim = grid;
            kp.blockDim = block;
            kp.sharedMemBytes = (unsigned)shmem;
            kp.kernelParams = ptrs;
            cudaGraphNode_t node;
            e = cudaGraphAddKernelNode(&node, graph, last ? &last : nullptr, last ? 1 : 0, &kp);
            last = node;
            ++nodes;
        } else {
            e = cudaLaunchKernel((const void*)kernel, grid, block, ptrs, shmem, stream);
            if (e == cudaSuccess) ++c->launches;
        }
        if (e != cudaSuccess) {
            c->cuda_err = (int)e;
            rc = LRMD_ECUDA;
            (void)cudaGetLastError();
        }
    }

    // The dominant kernel of the model: bracketed by CUDA events on the launching stream when
    // LRMD_OPT_KERNEL_TIMING is on (never inside a graph).
    template <typename... KA, typename... A>
    void go_timed(void (*kernel)(KA...), dim3 grid, dim3 block, A... a) {
        const bool t = c->timing && !graph && rc == LRMD_OK && c->ev_used + 2 <= kMaxTimedEvents;
        if (t) {
            while (c->ev.size() < c->ev_used + 2) {
                cudaEvent_t e;
                if (cudaEventCreate(&e) != cudaSuccess) { (void)cudaGetLastError(); go(kernel, grid, block, a...); return; }
                c->ev.push_back(e);
            }
            const cudaError_t e = cudaEventRecord(c->ev[c->ev_used], stream);
            if (e != cudaSuccess) { c->cuda_err = (int)e; rc = LRMD_ECUDA; (void)cudaGetLastError(); return; }
        }
        go(kernel, grid, block, a...);
        if (t) {
            const cudaError_t e = cudaEventRecord(c->ev[c->ev_used + 1], stream);
            if (e != cudaSuccess) { c->cuda_err = (int)e; rc = LRMD_ECUDA; (void)cudaGetLastError(); return; }
            c->ev_used += 2;
        }
    }

    template <typename T, size_t... I>
    static void fill(void** ptrs, T& vals, std::index_sequence<I...>) {
        ((ptrs[I] = (void*)&std::get<I>(vals)), ...);
    }
};

inline double2* hmf_buf(lrmd_ctx* c, int k) {
    return reinterpret_cast<double2*>(c->ws + c->lay.hmf_partial) + (size_t)k * kHmfMaxGrid;
}
inline bool is_sharded(const lrmd_ctx* c) { return c->N_total != c->N; }
inline double2* shared2_ptr(lrmd_ctx* c) { return reinterpret_cast<double2*>(c->ws + c->lay.shared2); }
// where the kernels read (sum cos, sum sin) from: the rank-summed pair of a shard, or the per-CTA partials
inline const double2* hmf_sums(lrmd_ctx* c, int buf) { return is_sharded(c) ? shared2_ptr(c) : hmf_buf(c, buf); }
inline int hmf_nsums(const lrmd_ctx* c) { return is_sharded(c) ? 1 : c->hmf_grid; }
inline double2* js_ptr(lrmd_ctx* c) { return reinterpret_cast<double2*>(c->ws + c->lay.js); }
inline float2* js32_ptr(lrmd_ctx* c) {
    return c->opt_precision == 1 ? reinterpret_cast<float2*>(c->ws + c->lay.js32) : nullptr;
}
inline double* part0(lrmd_ctx* c) { return reinterpret_cast<double*>(c->ws + c->lay.partial0); }
inline double* part1(lrmd_ctx* c) {
    return c->model == LRMD_GRAV2D ? reinterpret_cast<double*>(c->ws + c->lay.partial1) : nullptr;
}
inline double* kpart(lrmd_ctx* c) { return reinterpret_cast<double*>(c->ws + c->lay.kpart); }
inline double* vpart(lrmd_ctx* c) { return reinterpret_cast<double*>(c->ws + c->lay.vpart); }

struct Coef { double B0, B1, D0, D1; };
Coef coefficients() {
    // Yoshida's triple jump (reading G4): w1 = 1/(2 - 2^(1/3)), w0 = -2^(1/3)/(2 - 2^(1/3)).
    const double cb = std::cbrt(2.0);
    const double w1 = 1.0 / (2.0 - cb), w0 = -cb / (2.0 - cb);
    return Coef{0.5 * w1, 0.5 * (w0 + w1), w1, w0};
}

// ---- HMF sequencing ----------------------------------------------------------------------------------

// Launch the fused substage kernel of the context's variant with the given stage flags.
template <bool KICK, bool KICK2, bool DRIFT, bool REDUCE>
void hmf_launch(Launcher& L, bool timed, double kickA, double kickB, double drift, int in_buf, int out_buf) {
    lrmd_ctx* c = L.c;
    const dim3 g(c->hmf_grid);
    const double2* pin = hmf_sums(c, in_buf);
    const int gin = hmf_nsums(c);
    const double inv_n = 1.0 / (double)c->N_total;
    double2* pout = hmf_buf(c, out_buf);
#define LRMD_HMF_GO(KERNEL, BLOCK)                                                                           \
    do {                                                                                                     \
        if (timed) L.go_timed(KERNEL, g, dim3(BLOCK), c->a0, c->a1, c->N, inv_n, kickA, kickB, drift, pin, gin, pout); \
        else L.go(KERNEL, g, dim3(BLOCK), c->a0, c->a1, c->N, inv_n, kickA, kickB, drift, pin, gin, pout);     \
    } while (0)
#define LRMD_HMF_TMA(V, CONS, NS, MINB)                                                                      \
    case V:                                                                                                  \
        L.smem = HmfTma<CONS, NS>::kSmemBytes;                                                               \
        LRMD_HMF_GO((hmf_substage_tma_kernel<KICK, KICK2, DRIFT, REDUCE, CONS, NS, MINB>), CONS + 32);       \
        break
    switch (c->hmf_variant) {
        LRMD_HMF_TMA(1, 512, 4, 1);
        LRMD_HMF_TMA(2, 256, 6, 2);
        default:
            LRMD_HMF_GO((hmf_substage_kernel<KICK, KICK2, DRIFT, REDUCE>), kHmfThreads);
            break;
    }
#undef LRMD_HMF_TMA
#undef LRMD_HMF_GO
    if (REDUCE && is_sharded(c)) {
        // each GPU's contribution to the magnetisation, summed over the GPUs
        L.go(hmf_collapse_kernel, dim3(1), dim3(kHmfThreads), (const double2*)pout, c->hmf_grid, shared2_ptr(c));
        if (L.rc == LRMD_OK && c->allreduce && c->allreduce(shared2_ptr(c), 2, L.stream, c->coll_user) != 0) L.rc = LRMD_ECOLL;
    }
}

// One fused substage: [kick kickA (+kickB)] -> drift -> reduce into the next partial buffer.
void hmf_substage(Launcher& L, bool kick2, double kickA, double kickB, double drift, int& cur) {
    const int nxt = (cur + 1) % 3;
    if (kick2) hmf_launch<true, true, true, true>(L, true, kickA, kickB, drift, cur, nxt);
    else hmf_launch<true, false, true, true>(L, true, kickA, 0.0, drift, cur, nxt);
    cur = nxt;
}

void hmf_reduce_only(Launcher& L) {
    hmf_launch<false, false, false, true>(L, false, 0.0, 0.0, 0.0, L.c->cur, L.c->cur);
}

// One full step.  merged: the closing kick B0 dt of the previous step is folded into this
// step's first substage (same force, two FMAs in the order they would have run separately).
void hmf_one_step(Launcher& L, const Coef& k, double dt, bool merged, int& cur) {
    hmf_substage(L, merged, k.B0 * dt, k.B0 * dt, k.D0 * dt, cur);
    hmf_substage(L, false, k.B1 * dt, 0.0, k.D1 * dt, cur);
    hmf_substage(L, false, k.B1 * dt, 0.0, k.D0 * dt, cur);
}

void hmf_closing_kick(Launcher& L, const Coef& k, double dt, int cur) {
    hmf_launch<true, false, false, false>(L, false, k.B0 * dt, 0.0, 0.0, cur, cur);
}

int hmf_build_graph(lrmd_ctx* c, const Coef& k, double dt) {
    drop_graph(c);
    cudaGraph_t g;
    cudaError_t e = cudaGraphCreate(&g, 0);
    if (e != cudaSuccess) { c->cuda_err = (int)e; return LRMD_ECUDA; }
    Launcher L{c, nullptr};
    L.graph = g;
    int cur = c->cur;
    for (int s = 0; s < kGraphSteps; ++s) hmf_one_step(L, k, dt, true, cur);
    int rc = L.rc;
    if (rc == LRMD_OK) {
        e = cudaGraphInstantiate(&c->graph_exec, g, 0);
        if (e != cudaSuccess) { c->cuda_err = (int)e; rc = LRMD_ECUDA; c->graph_exec = nullptr; }
    }
    cudaGraphDestroy(g);
    if (rc == LRMD_OK) { c->graph_dt = dt; c->graph_cur = c->cur; c->graph_nodes = L.nodes; }
    return rc;
}

// All n steps in one launch of one thread-block cluster (hmf_cluster_kernel).
int hmf_step_cluster(lrmd_ctx* c, int64_t n, double dt, cudaStream_t stream) {
    const Coef k = coefficients();
    const int ctas = c->hmf_grid;     // 8, or 16 when the device grants the non-portable cluster size
    const int64_t per = (int64_t)ctas * kHmfClusterThreads;
    const int P = c->N <= per ? 1 : (c->N <= 2 * per ? 2 : (c->N <= 4 * per ? 4 : 8));
    void (*kernel)(double*, double*, long long, long long, double, double, double, double, double2*) =
        P == 1 ? hmf_cluster_kernel<1> : (P == 2 ? hmf_cluster_kernel<2> : (P == 4 ? hmf_cluster_kernel<4> : hmf_cluster_kernel<8>));
    if (ctas > kHmfClusterCtas) {
        bool ready = false;
        for (const void* f : c->smem_ready) ready = ready || f == (const void*)kernel;
        if (!ready) {
            const cudaError_t ea = cudaFuncSetAttribute((const void*)kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
            if (ea != cudaSuccess) { c->cuda_err = (int)ea; (void)cudaGetLastError(); return LRMD_ECUDA; }
            c->smem_ready.push_back((const void*)kernel);
        }
    }
    cudaLaunchConfig_t cfg;
    std::memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3(ctas);
    cfg.blockDim = dim3(kHmfClusterThreads);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = ctas;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    const bool t = c->timing && c->ev_used + 2 <= kMaxTimedEvents;
    if (t) {
        while (c->ev.size() < c->ev_used + 2) {
            cudaEvent_t e;
            const cudaError_t ee = cudaEventCreate(&e);
            if (ee != cudaSuccess) { c->cuda_err = (int)ee; (void)cudaGetLastError(); return LRMD_ECUDA; }
            c->ev.push_back(e);
        }
        cudaEventRecord(c->ev[c->ev_used], stream);
    }
    const cudaError_t e = cudaLaunchKernelEx(&cfg, kernel, c->a0, c->a1, (long long)c->N, (long long)n, k.B0 * dt,
                                             k.B1 * dt, k.D0 * dt, k.D1 * dt, hmf_buf(c, c->cur));
    if (e != cudaSuccess) { c->cuda_err = (int)e; (void)cudaGetLastError(); return LRMD_ECUDA; }
    if (t) { cudaEventRecord(c->ev[c->ev_used + 1], stream); c->ev_used += 2; }
    ++c->launches;
    c->force_valid = true;   // the kernel leaves the sums at the final angles in the current partial buffer
    return LRMD_OK;
}

// Errors that mean "this device will not run the grid-resident kernel" (too few SMs for one CTA each, no cooperative
// launch, shared memory not granted); anything else is a real failure and is reported as LRMD_ECUDA.
inline bool grid_refused(cudaError_t e) {
    return e == cudaErrorCooperativeLaunchTooLarge || e == cudaErrorNotSupported || e == cudaErrorInvalidValue ||
           e == cudaErrorInvalidConfiguration;
}

// All n steps in one cooperative launch of one CTA per SM (hmf_grid_kernel).  Returns LRMD_EUNSUPPORTED if the device
// refuses the cooperative launch (the caller then falls back to the substage kernels).
int hmf_step_grid(lrmd_ctx* c, int64_t n, double dt, cudaStream_t stream) {
    const Coef k = coefficients();
    const int G = c->hmf_grid;
    const int nlocal = (int)((c->N + G - 1) / G);
    const size_t smem = (size_t)nlocal * kHmfGridBytesPerParticle;
    bool ready = false;
    for (const void* f : c->smem_ready) ready = ready || f == (const void*)hmf_grid_kernel;
    if (!ready) {
        const cudaError_t ea = cudaFuncSetAttribute((const void*)hmf_grid_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                    (int)((size_t)kHmfGridMaxLocal * kHmfGridBytesPerParticle));
        if (ea != cudaSuccess) { c->cuda_err = (int)ea; (void)cudaGetLastError(); return grid_refused(ea) ? LRMD_EUNSUPPORTED : LRMD_ECUDA; }
        c->smem_ready.push_back((const void*)hmf_grid_kernel);
    }
    cudaLaunchConfig_t cfg;
    std::memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3(G);
    cfg.blockDim = dim3(kHmfGridThreads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeCooperative;
    attr[0].val.cooperative = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    const bool t = c->timing && c->ev_used + 2 <= kMaxTimedEvents;
    if (t) {
        while (c->ev.size() < c->ev_used + 2) {
            cudaEvent_t e;
            const cudaError_t ee = cudaEventCreate(&e);
            if (ee != cudaSuccess) { c->cuda_err = (int)ee; (void)cudaGetLastError(); return LRMD_ECUDA; }
            c->ev.push_back(e);
        }
        cudaEventRecord(c->ev[c->ev_used], stream);
    }
    const int nxt = (c->cur + 1) % 3;
    const cudaError_t e = cudaLaunchKernelEx(&cfg, hmf_grid_kernel, c->a0, c->a1, (long long)c->N, nlocal, (long long)n,
                                             k.B0 * dt, k.B1 * dt, k.D0 * dt, k.D1 * dt, hmf_buf(c, nxt), hmf_buf(c, c->cur));
    if (e != cudaSuccess) { c->cuda_err = (int)e; (void)cudaGetLastError(); return grid_refused(e) ? LRMD_EUNSUPPORTED : LRMD_ECUDA; }
    if (t) { cudaEventRecord(c->ev[c->ev_used + 1], stream); c->ev_used += 2; }
    ++c->launches;
    c->force_valid = true;   // the kernel leaves the per-CTA sums at the final angles in the current partial buffer
    return LRMD_OK;
}

int hmf_step(lrmd_ctx* c, int64_t n, double dt, cudaStream_t stream) {
    if (c->hmf_variant == kHmfClusterVariant) return hmf_step_cluster(c, n, dt, stream);
    if (c->hmf_variant == kHmfGridVariant) {
        const int rc = hmf_step_grid(c, n, dt, stream);
        if (rc != LRMD_EUNSUPPORTED) return rc;
        // the device does not grant the cooperative launch (fewer SMs available than CTAs): substage kernels instead
        c->grid_unavailable = true;
        resolve(c);
        drop_graph(c);
        c->force_valid = false;
    }
    const Coef k = coefficients();
    Launcher L{c, stream};
    if (!c->force_valid) { hmf_reduce_only(L); c->force_valid = true; }
    int cur = c->cur;
    hmf_one_step(L, k, dt, false, cur);     // cur returns to c->cur after 3 substages
    int64_t left = n - 1;
    if (L.rc != LRMD_OK) return L.rc;
    if (c->use_graph && !c->timing && left >= kGraphSteps) {
        cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
        cudaStreamIsCapturing(stream, &cs);
        if (cs == cudaStreamCaptureStatusNone) {
            if (!c->graph_exec || c->graph_dt != dt || c->graph_cur != c->cur) {
                const int rc = hmf_build_graph(c, k, dt);
                if (rc != LRMD_OK) return rc;
            }
            while (left >= kGraphSteps) {
                const cudaError_t e = cudaGraphLaunch(c->graph_exec, stream);
                if (e != cudaSuccess) { c->cuda_err = (int)e; (void)cudaGetLastError(); return LRMD_ECUDA; }
                c->launches += c->graph_nodes;
                left -= kGraphSteps;
            }
        }
    }
    for (; left > 0; --left) hmf_one_step(L, k, dt, true, cur);
    hmf_closing_kick(L, k, dt, cur);
    return L.rc;
}

// ---- pair-model sequencing ---------------------------------------------------------------------------

// Shards: every rank needs all positions for its rows' pair sums ("each GPU holds all
// positions"; the paper copies halves peer to peer, here the caller's all-gather fills the packed stream in place).
void pair_gather(Launcher& L) {
    lrmd_ctx* c = L.c;
    if (!is_sharded(c) || !c->allgather || L.rc != LRMD_OK) return;
    if (c->allgather(js_ptr(c), (int64_t)sizeof(double2), c->i0, c->N, c->N_total, L.stream, c->coll_user) != 0) L.rc = LRMD_ECOLL;
    if (L.rc == LRMD_OK && js32_ptr(c) &&
        c->allgather(js32_ptr(c), (int64_t)sizeof(float2), c->i0, c->N, c->N_total, L.stream, c->coll_user) != 0)
        L.rc = LRMD_ECOLL;
}

void pair_pack(Launcher& L) {
    lrmd_ctx* c = L.c;
    const dim3 g((unsigned)((c->N + kUpdThreads - 1) / kUpdThreads)), b(kUpdThreads);
    if (c->model == LRMD_RING)
        L.go(pair_pack_kernel<1>, g, b, c->a0, (const double*)nullptr, c->N, c->i0, js_ptr(c), js32_ptr(c));
    else L.go(pair_pack_kernel<2>, g, b, c->a0, c->a1, c->N, c->i0, js_ptr(c), js32_ptr(c));
    pair_gather(L);
}

inline double* wsd(lrmd_ctx* c, size_t off) { return off ? reinterpret_cast<double*>(c->ws + off) : nullptr; }

// Symmetric force evaluation (row N4): per batch of tiles one kernel launch + the fold into the force row.
// upd: 0 = none, 1 kick, 2 kick + drift, 3 two kicks + drift, fused into the fold (single-launch evaluations only;
// the caller checks pair_can_fuse).
void pair_force_sym(Launcher& L, int upd = 0, double kickA = 0.0, double kickB = 0.0, double drift = 0.0) {
    lrmd_ctx* c = L.c;
    double *i0 = wsd(c, c->lay.ipart0), *i1 = wsd(c, c->lay.ipart1), *j0 = wsd(c, c->lay.jpart0), *j1 = wsd(c, c->lay.jpart1);
    const double pre = c->model == LRMD_RING ? -1.0 / (2.0 * std::sqrt(2.0) * (double)c->N) : -2.0 / (double)c->N;
    for (const int4& bt : c->sym_batches) {
        SymPart S = c->spart;
        S.tile0 = bt.x; S.tile1 = bt.y; S.w0 = bt.z; S.G = bt.w;
        const dim3 g((unsigned)((S.G + kSymThreads / 32 - 1) / (kSymThreads / 32))), b(kSymThreads);
        if (c->opt_precision == 1) {
            if (c->sym_R == 8) L.go_timed(grav_force_sym_f32_kernel<8>, g, b, (const float2*)js32_ptr(c), S, (float)c->eps, pre, i0, i1, j0, j1);
            else L.go_timed(grav_force_sym_f32_kernel<4>, g, b, (const float2*)js32_ptr(c), S, (float)c->eps, pre, i0, i1, j0, j1);
        } else {
#define LRMD_SYM_GO(M, RR, X, MB) L.go_timed(pair_force_sym_kernel<M, RR, X, MB>, g, b, js_ptr(c), S, c->eps, pre, i0, i1, j0, j1)
#define LRMD_SYM_X(M, RR)                                   \
            switch (c->sym_xch) {                           \
                case 0: LRMD_SYM_GO(M, RR, 0, 2); break;    \
                case 1: LRMD_SYM_GO(M, RR, 1, 2); break;    \
                case 2: LRMD_SYM_GO(M, RR, 1, 3); break;    \
                default: LRMD_SYM_GO(M, RR, 1, 4); break;   \
            }
            if (c->model == LRMD_RING) {
                if (c->sym_R == 8) { LRMD_SYM_X(1, 8) } else { LRMD_SYM_X(1, 4) }
            } else {
                if (c->sym_R == 8) { LRMD_SYM_X(2, 8) } else { LRMD_SYM_X(2, 4) }
            }
#undef LRMD_SYM_X
#undef LRMD_SYM_GO
        }
        // rows of this batch only concern particles from its first tile on
        const long long first = (long long)S.tile0 * S.T;
        FusedUpdate U;
        U.q0 = c->a0; U.q1 = nullptr; U.p0 = c->a1; U.p1 = nullptr;
        if (c->model == LRMD_GRAV2D) { U.q1 = c->a1; U.p0 = c->a2; U.p1 = c->a3; }
        U.kickA = kickA; U.kickB = kickB; U.drift = drift; U.js = js_ptr(c); U.js32 = js32_ptr(c);
        const dim3 fg((unsigned)((c->N - first + 31) / 32)), fb(32, kFoldGroups);
#define LRMD_FOLD(M, UPD) \
        L.go(pair_sym_fold_kernel<M, UPD>, fg, fb, S, (const double*)i0, (const double*)i1, (const double*)j0, \
             (const double*)j1, part0(c), part1(c), U)
        if (c->model == LRMD_RING) {
            if (upd == 1) LRMD_FOLD(1, 1); else if (upd == 2) LRMD_FOLD(1, 2); else if (upd == 3) LRMD_FOLD(1, 3); else LRMD_FOLD(1, 0);
        } else {
            if (upd == 1) LRMD_FOLD(2, 1); else if (upd == 2) LRMD_FOLD(2, 2); else if (upd == 3) LRMD_FOLD(2, 3); else LRMD_FOLD(2, 0);
        }
#undef LRMD_FOLD
    }
}

// Band-kernel force evaluation: one launch + the fold (which takes the update that follows, upd as above).
void pair_force_band(Launcher& L, int upd = 0, double kickA = 0.0, double kickB = 0.0, double drift = 0.0, bool withv = false) {
    lrmd_ctx* c = L.c;
    // V = pre_v * sum_{i<j} t_ij (eqs.(1),(3)), delivered with the force when withv
    const double pre_v = c->model == LRMD_RING ? -1.0 / (std::sqrt(2.0) * (double)c->N) : 1.0 / (double)c->N;
    double *i0 = wsd(c, c->lay.bibuf0), *i1 = wsd(c, c->lay.bibuf1), *j0 = wsd(c, c->lay.bjbuf0), *j1 = wsd(c, c->lay.bjbuf1);
    const double pre = c->model == LRMD_RING ? -1.0 / (2.0 * std::sqrt(2.0) * (double)c->N) : -2.0 / (double)c->N;
    const dim3 g((unsigned)c->bpart.P), b(kBandThreads);
    if (c->opt_precision == 1) {
        L.smem = band_f32_smem_bytes(c->band_R);
#define LRMD_BAND32_GO(RR, X) L.go_timed(grav_force_band_f32_kernel<RR, X>, g, b, (const float2*)js32_ptr(c), c->bpart, (float)c->eps, pre, i0, i1, j0, j1)
        // LRMD_OPT_PAIR_SYM_EXCHANGE 0 / -1 (default): the j-side fp32 packet travels by shuffles, one fp64 add per chunk
        // visit (11 % faster at N = 2^20 than 1-3, the per-step shared-memory exchange; worst error 4e-8 A_i either way)
        const bool jshfl = c->opt_sym_xch <= 0;
        if (c->band_R == 16) { if (jshfl) LRMD_BAND32_GO(16, true); else LRMD_BAND32_GO(16, false); }
        else if (c->band_R == 8) { if (jshfl) LRMD_BAND32_GO(8, true); else LRMD_BAND32_GO(8, false); }
        else { if (jshfl) LRMD_BAND32_GO(4, true); else LRMD_BAND32_GO(4, false); }
#undef LRMD_BAND32_GO
        withv = false;
    } else {
    L.smem = band_smem_bytes(c->band_R);
#define LRMD_BAND_GO(M, RR, V) \
    L.go_timed(pair_force_band_kernel<M, RR, V>, g, b, (const double2*)js_ptr(c), c->bpart, c->eps, pre, i0, i1, j0, j1, pre_v, vpart(c))
#define LRMD_BAND_V(M, RR) do { if (withv) LRMD_BAND_GO(M, RR, true); else LRMD_BAND_GO(M, RR, false); } while (0)
    if (c->model == LRMD_RING) {
        if (c->band_R == 8) LRMD_BAND_V(1, 8); else LRMD_BAND_V(1, 4);
    } else {
        if (c->band_R == 8) LRMD_BAND_V(2, 8); else LRMD_BAND_V(2, 4);
    }
#undef LRMD_BAND_V
#undef LRMD_BAND_GO
    }
    c->v_valid = withv;
    FusedUpdate U;
    U.q0 = c->a0; U.q1 = nullptr; U.p0 = c->a1; U.p1 = nullptr;
    if (c->model == LRMD_GRAV2D) { U.q1 = c->a1; U.p0 = c->a2; U.p1 = c->a3; }
    U.kickA = kickA; U.kickB = kickB; U.drift = drift; U.js = js_ptr(c); U.js32 = js32_ptr(c);
    const dim3 fg((unsigned)((c->N + 31) / 32)), fb(32, kFoldGroups);
#define LRMD_BFOLD(M, UPD) \
    L.go(pair_band_fold_kernel<M, UPD>, fg, fb, c->bpart, (const double*)i0, (const double*)i1, (const double*)j0, \
         (const double*)j1, part0(c), part1(c), U)
    if (c->model == LRMD_RING) {
        if (upd == 1) LRMD_BFOLD(1, 1); else if (upd == 2) LRMD_BFOLD(1, 2); else if (upd == 3) LRMD_BFOLD(1, 3); else LRMD_BFOLD(1, 0);
    } else {
        if (upd == 1) LRMD_BFOLD(2, 1); else if (upd == 2) LRMD_BFOLD(2, 2); else if (upd == 3) LRMD_BFOLD(2, 3); else LRMD_BFOLD(2, 0);
    }
#undef LRMD_BFOLD
}

ForceRows force_rows(lrmd_ctx* c) {
    ForceRows FR;
    FR.partial0 = part0(c);
    FR.partial1 = part1(c);
    FR.single_row = c->sym ? 1 : 0;
    return FR;
}

void pair_force(Launcher& L, bool withv = false) {
    lrmd_ctx* c = L.c;
    if (c->band) { pair_force_band(L, 0, 0.0, 0.0, 0.0, withv); return; }
    if (c->sym) { pair_force_sym(L); return; }
    with_pair_cfg(c->pair_variant, [&](auto cfg) {
        using CFG = decltype(cfg);
        const dim3 g((unsigned)c->part.G), b(CFG::THREADS);
        if (c->model == LRMD_RING && c->opt_precision == 1)
            L.go_timed(ring_force_f32_kernel<CFG>, g, b, (const float2*)js32_ptr(c), c->part, (float)c->eps,
                       -1.0 / (2.0 * std::sqrt(2.0) * (double)c->N_total), part0(c));
        else if (c->model == LRMD_RING)
            L.go_timed(pair_force_kernel<1, CFG>, g, b, js_ptr(c), c->part, c->eps,
                       -1.0 / (2.0 * std::sqrt(2.0) * (double)c->N_total), part0(c), part1(c));
        else if (c->opt_precision == 1)
            L.go_timed(grav_force_f32_kernel<CFG>, g, b, (const float2*)js32_ptr(c), c->part, (float)c->eps,
                       -2.0 / (double)c->N_total, part0(c), part1(c));
        else
            L.go_timed(pair_force_kernel<2, CFG>, g, b, js_ptr(c), c->part, c->eps, -2.0 / (double)c->N_total, part0(c),
                       part1(c));
    });
}

void pair_update(Launcher& L, bool kick2, bool drift, double kickA, double kickB, double d) {
    lrmd_ctx* c = L.c;
    const dim3 g((unsigned)((c->N + kUpdThreads - 1) / kUpdThreads)), b(kUpdThreads);
    double *q0 = c->a0, *q1 = nullptr, *p0 = c->a1, *p1 = nullptr;
    if (c->model == LRMD_GRAV2D) { q1 = c->a1; p0 = c->a2; p1 = c->a3; }
#define LRMD_UPD(M, K2, DR) \
    L.go(pair_update_kernel<M, K2, DR>, g, b, q0, q1, p0, p1, c->part, force_rows(c), kickA, kickB, d, js_ptr(c), js32_ptr(c))
    if (c->model == LRMD_RING) {
        if (!drift) LRMD_UPD(1, false, false);
        else if (kick2) LRMD_UPD(1, true, true);
        else LRMD_UPD(1, false, true);
    } else {
        if (!drift) LRMD_UPD(2, false, false);
        else if (kick2) LRMD_UPD(2, true, true);
        else LRMD_UPD(2, false, true);
    }
#undef LRMD_UPD
    if (drift) pair_gather(L);   // the packed stream changed: every rank needs the new positions
}

void pair_ensure_force(Launcher& L) {
    lrmd_ctx* c = L.c;
    if (!c->js_valid) { pair_pack(L); c->js_valid = true; }
    if (!c->force_valid) { pair_force(L); c->force_valid = true; }
}

int pair_step(lrmd_ctx* c, int64_t n, double dt, cudaStream_t stream) {
    const Coef k = coefficients();
    Launcher L{c, stream};
    pair_ensure_force(L);
    // A force evaluation that is one launch of the symmetric kernel takes the update that follows it into its
    // fold kernel (same arithmetic, one launch and one pass over the force row fewer per substage).
    const bool fuse = (c->band || (c->sym && c->sym_batches.size() == 1)) && c->opt_fuse != 0;
    auto force_then_update = [&](bool kick2, bool drift, double kA, double kB, double d, bool withv = false) {
        if (fuse) {
            if (c->band) pair_force_band(L, drift ? (kick2 ? 3 : 2) : 1, kA, kB, d, withv);
            else pair_force_sym(L, drift ? (kick2 ? 3 : 2) : 1, kA, kB, d);
        } else {
            pair_force(L, withv);
            pair_update(L, kick2, drift, kA, kB, d);
        }
    };
    c->v_valid = false;
    pair_update(L, false, true, k.B0 * dt, 0.0, k.D0 * dt);
    for (int64_t s = 0; s < n; ++s) {
        force_then_update(false, true, k.B1 * dt, 0.0, k.D1 * dt);
        force_then_update(false, true, k.B1 * dt, 0.0, k.D0 * dt);
        if (s + 1 < n) force_then_update(true, true, k.B0 * dt, k.B0 * dt, k.D0 * dt);   // closing + opening kick
        else force_then_update(false, false, k.B0 * dt, 0.0, 0.0, c->band && c->want_v);   // closing kick (+ V for a record)
    }
    return L.rc;
}

bool finite_pos(double x) { return std::isfinite(x) && x > 0.0; }

}  // namespace

// ---- lrmd_hmf_forces_static: the one call whose scratch is built into the library --------------------
// For callers that cannot hand over a workspace (see include/lrmd.h).  The per-CTA (sum cos, sum sin) pairs of the
// reduction go to the file-scope array below instead of the caller's workspace: 4096 pairs = 64 KiB, resident on every
// GPU that loads the library.  One CTA sums a fixed block of 1024 particles, so the number of CTAs — and with it the
// scratch — grows with N; 4096 CTAs cover LRMD_STATIC_MAX_N particles and a larger N is refused.
constexpr int kStaticMaxCtas = 4096;
constexpr int kStaticPerThread = 4;
constexpr int kStaticPerCta = kStaticPerThread * lrmd::kHmfThreads;   // 1024
constexpr int kStaticMaxDevices = 64;
static_assert((long long)kStaticMaxCtas * kStaticPerCta == LRMD_STATIC_MAX_N, "lrmd.h states this limit");
static_assert(sizeof(double2) * kStaticMaxCtas == LRMD_STATIC_SCRATCH_BYTES, "lrmd.h states this size");

static __device__ __align__(256) double2 g_lrmd_static_partials[kStaticMaxCtas];

// Variant of the reduce-only substage kernel (hmf_substage_kernel<false, false, false, true>): same per-particle
// arithmetic and the same fixed block-sum tree, but CTA b always owns particles [1024 b, 1024 b + 1024) (no grid
// stride, scalar loads: theta needs 8-byte alignment only) and writes its pair to partial_out[b], which the host passes
// as the device address of g_lrmd_static_partials.  Every entry the force kernel reads afterwards (0 .. gridDim.x - 1)
// is written here first, so the array never needs clearing.
__global__ void __launch_bounds__(lrmd::kHmfThreads)
hmf_reduce_static_kernel(const double* __restrict__ theta, long long N, double2* __restrict__ partial_out) {
    __shared__ double scratch[2 * (lrmd::kHmfThreads / 32)];
    const long long base = (long long)blockIdx.x * kStaticPerCta + threadIdx.x;
    double r[2] = {0.0, 0.0};
#pragma unroll
    for (int k = 0; k < kStaticPerThread; ++k) {
        const long long i = base + (long long)k * lrmd::kHmfThreads;
        if (i < N) {
            double s, c;
            lrmd::sincos_any(theta[i], s, c);
            r[0] += c;
            r[1] += s;
        }
    }
    lrmd::block_sum<lrmd::kHmfThreads, 2>(r, scratch);
    if (threadIdx.x == 0) partial_out[blockIdx.x] = make_double2(r[0], r[1]);
}

namespace {

// Device address of g_lrmd_static_partials on the current device.  In host code the array's name stands for a host-side
// shadow object, not for device memory, so the address is asked for once per device (with that device current) and
// kept.  cudaGetSymbolAddress allocates nothing: the array is part of the loaded module.
std::mutex g_static_mutex;
double2* g_static_addr[kStaticMaxDevices] = {};

int static_partials(double2** out, cudaError_t* err) {
    int dev = -1;
    *err = cudaGetDevice(&dev);
    if (*err != cudaSuccess) { (void)cudaGetLastError(); return LRMD_ECUDA; }
    if (dev < 0 || dev >= kStaticMaxDevices) return LRMD_EUNSUPPORTED;
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_addr[dev]) {
        void* p = nullptr;
        *err = cudaGetSymbolAddress(&p, g_lrmd_static_partials);
        if (*err != cudaSuccess || !p) {
            (void)cudaGetLastError();
            if (*err == cudaSuccess) *err = cudaErrorInvalidSymbol;
            return LRMD_ECUDA;
        }
        g_static_addr[dev] = static_cast<double2*>(p);
    }
    *out = g_static_addr[dev];
    return LRMD_OK;
}

}  // namespace

// =========================================== C ABI =====================================================

extern "C" {

int lrmd_create(lrmd_ctx** out, int model, int64_t N, double eps) {
    if (!out) return LRMD_EINVAL;
    *out = nullptr;
    if (model < LRMD_HMF || model > LRMD_GRAV2D || N < 1) return LRMD_EINVAL;
    if (N > ((int64_t)1 << 40)) return LRMD_EINVAL;
    if (model != LRMD_HMF && N > ((int64_t)1 << 28)) return LRMD_EINVAL;   // O(N^2) models: 7e16 pairs per force
    if (model != LRMD_HMF && !finite_pos(eps)) return LRMD_EINVAL;
    lrmd_ctx* c = new (std::nothrow) lrmd_ctx();
    if (!c) return LRMD_ESTATE;     // host allocation failed: there is no context to report on
    c->model = model;
    c->N = N;
    c->N_total = N;
    c->eps = (model == LRMD_HMF) ? 0.0 : eps;
    resolve(c);
    *out = c;
    return LRMD_OK;
}

int lrmd_destroy(lrmd_ctx* c) {
    if (!c) return LRMD_EINVAL;
    drop_graph(c);
    for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
    delete c;
    return LRMD_OK;
}

int lrmd_workspace_bytes(const lrmd_ctx* c, size_t* bytes) {
    if (!c || !bytes) return LRMD_EINVAL;
    *bytes = c->lay.total;
    return LRMD_OK;
}

int lrmd_set_workspace(lrmd_ctx* c, void* device_ptr, size_t bytes, void* cuda_stream) {
    // every buffer is written by a kernel before it is read, except the two small work tables of the symmetric
    // pair kernel, which are copied here (host -> device on the given stream)
    if (!c || !device_ptr) return LRMD_EINVAL;
    if (bytes < c->lay.total || ((uintptr_t)device_ptr % kAlign) != 0) return LRMD_EINVAL;
    c->ws = static_cast<char*>(device_ptr);
    if (c->band) {
        cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
        cudaError_t e = cudaMemcpyAsync(c->ws + c->lay.band_wpiece, c->band_wpiece.data(), sizeof(int) * c->band_wpiece.size(),
                                        cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess)
            e = cudaMemcpyAsync(c->ws + c->lay.band_pieces, c->band_pieces.data(), sizeof(BandPiece) * c->band_pieces.size(),
                                cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess)
            e = cudaMemcpyAsync(c->ws + c->lay.band_infos, c->band_infos.data(), sizeof(BandInfo) * c->band_infos.size(),
                                cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) { c->cuda_err = (int)e; (void)cudaGetLastError(); c->ws = nullptr; return LRMD_ECUDA; }
        c->bpart.wpiece = reinterpret_cast<const int*>(c->ws + c->lay.band_wpiece);
        c->bpart.pieces = reinterpret_cast<const BandPiece*>(c->ws + c->lay.band_pieces);
        c->bpart.bands = reinterpret_cast<const BandInfo*>(c->ws + c->lay.band_infos);
    }
    if (c->sym) {
        cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
        cudaError_t e = cudaMemcpyAsync(c->ws + c->lay.sym_wstart, c->sym_wstart.data(), sizeof(int4) * c->sym_wstart.size(),
                                        cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess)
            e = cudaMemcpyAsync(c->ws + c->lay.sym_tiles, c->sym_tiles.data(), sizeof(int2) * c->sym_tiles.size(),
                                cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);    // the host vectors may change after this call
        if (e != cudaSuccess) { c->cuda_err = (int)e; (void)cudaGetLastError(); c->ws = nullptr; return LRMD_ECUDA; }
        c->spart.wstart = reinterpret_cast<const int4*>(c->ws + c->lay.sym_wstart);
        c->spart.tile_rng = reinterpret_cast<const int2*>(c->ws + c->lay.sym_tiles);
    }
    c->force_valid = false;
    c->v_valid = false;
    c->js_valid = false;
    drop_graph(c);
    return LRMD_OK;
}

int lrmd_set_state(lrmd_ctx* c, double* a0, double* a1, double* a2, double* a3) {
    if (!c || !a0 || !a1) return LRMD_EINVAL;
    const bool two = c->model == LRMD_GRAV2D;
    if (two ? (!a2 || !a3) : (a2 || a3)) return LRMD_EINVAL;
    double* arr[4] = {a0, a1, a2, a3};
    for (double* p : arr)
        if (p && ((uintptr_t)p % 16) != 0) return LRMD_EINVAL;
    // the HMF kernel uses 256-bit accesses on theta and p
    if (c->model == LRMD_HMF && ((((uintptr_t)a0) % 32) != 0 || (((uintptr_t)a1) % 32) != 0)) return LRMD_EINVAL;
    c->a0 = a0; c->a1 = a1; c->a2 = a2; c->a3 = a3;
    c->state_set = true;
    c->force_valid = false;
    c->v_valid = false;
    c->js_valid = false;
    drop_graph(c);
    return LRMD_OK;
}

static int ready(const lrmd_ctx* c) {
    if (!c) return LRMD_EINVAL;
    if (!c->state_set || !c->ws) return LRMD_ESTATE;
    return LRMD_OK;
}

int lrmd_step(lrmd_ctx* c, int64_t n, double dt, void* cuda_stream) {
    int rc = ready(c);
    if (rc != LRMD_OK) return rc;
    if (n < 0 || !std::isfinite(dt)) return LRMD_EINVAL;
    if (n == 0) return LRMD_OK;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    return c->model == LRMD_HMF ? hmf_step(c, n, dt, stream) : pair_step(c, n, dt, stream);
}

int lrmd_step_host(lrmd_ctx* c, double* h0, double* h1, double* h2, double* h3, int64_t n, double dt,
                   void* cuda_stream) {
    int rc = ready(c);
    if (rc != LRMD_OK) return rc;
    const bool two = c->model == LRMD_GRAV2D;
    if (!h0 || !h1 || (two ? (!h2 || !h3) : (h2 || h3))) return LRMD_EINVAL;
    if (n < 0 || !std::isfinite(dt)) return LRMD_EINVAL;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    double* host[4] = {h0, h1, h2, h3};
    double* dev[4] = {c->a0, c->a1, c->a2, c->a3};
    const size_t bytes = sizeof(double) * (size_t)c->N;
    const int narr = two ? 4 : 2;
    cudaError_t e = cudaSuccess;
    for (int k = 0; k < narr && e == cudaSuccess; ++k)
        e = cudaMemcpyAsync(dev[k], host[k], bytes, cudaMemcpyHostToDevice, stream);
    if (e != cudaSuccess) { c->cuda_err = (int)e; (void)cudaGetLastError(); return LRMD_ECUDA; }
    c->force_valid = false;
    c->v_valid = false;
    c->js_valid = false;
    if (n > 0) {
        rc = c->model == LRMD_HMF ? hmf_step(c, n, dt, stream) : pair_step(c, n, dt, stream);
        if (rc != LRMD_OK) return rc;
    }
    for (int k = 0; k < narr && e == cudaSuccess; ++k)
        e = cudaMemcpyAsync(host[k], dev[k], bytes, cudaMemcpyDeviceToHost, stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
    if (e != cudaSuccess) { c->cuda_err = (int)e; (void)cudaGetLastError(); return LRMD_ECUDA; }
    return LRMD_OK;
}

int lrmd_forces(lrmd_ctx* c, double* f0, double* f1, void* cuda_stream) {
    int rc = ready(c);
    if (rc != LRMD_OK) return rc;
    if (!f0) return LRMD_EINVAL;
    if (c->model == LRMD_GRAV2D ? !f1 : (f1 != nullptr)) return LRMD_EINVAL;
    Launcher L{c, static_cast<cudaStream_t>(cuda_stream)};
    if (c->model == LRMD_HMF) {
        if (!c->force_valid) { hmf_reduce_only(L); c->force_valid = true; }
        int64_t g = (c->N + kHmfThreads - 1) / kHmfThreads;
        if (g > kHmfMaxGrid) g = kHmfMaxGrid;
        L.go(hmf_force_kernel, dim3((unsigned)g), dim3(kHmfThreads), (const double*)c->a0, f0, c->N,
             1.0 / (double)c->N_total, hmf_sums(c, c->cur), hmf_nsums(c));
    } else {
        pair_ensure_force(L);
        L.go(pair_force_out_kernel, dim3((unsigned)((c->N + kUpdThreads - 1) / kUpdThreads)), dim3(kUpdThreads), c->part,
             force_rows(c), f0, f1);
    }
    return L.rc;
}

int lrmd_energy(lrmd_ctx* c, double* out4_device, void* cuda_stream) {
    int rc = ready(c);
    if (rc != LRMD_OK) return rc;
    if (!out4_device) return LRMD_EINVAL;
    Launcher L{c, static_cast<cudaStream_t>(cuda_stream)};
    const bool two = c->model == LRMD_GRAV2D;
    const double* p0 = two ? c->a2 : c->a1;
    const double* p1 = two ? c->a3 : nullptr;
    int64_t gk = (c->N + kHmfThreads - 1) / kHmfThreads;
    if (gk > kEnergyGrid) gk = kEnergyGrid;
    L.go(kinetic_partial_kernel, dim3((unsigned)gk), dim3(kHmfThreads), p0, p1, c->N, kpart(c));
    if (c->model == LRMD_HMF) {
        if (!c->force_valid) { hmf_reduce_only(L); c->force_valid = true; }
        L.go(energy_finalize_kernel, dim3(1), dim3(kHmfThreads), c->model, c->N_total, (const double*)kpart(c), (int)gk,
             hmf_sums(c, c->cur), hmf_nsums(c), (const double*)nullptr, 0, out4_device);
    } else {
        if (!c->js_valid) { pair_pack(L); c->js_valid = true; }
        if (c->band && c->v_valid && c->force_valid) {
            // the force evaluation that ended the last step delivered V (lrmd_step_observe): no O(N^2) sweep
            L.go(energy_finalize_kernel, dim3(1), dim3(kHmfThreads), c->model, c->N, (const double*)kpart(c), (int)gk,
                 (const double2*)nullptr, 0, (const double*)vpart(c), c->bpart.P, out4_device);
            return L.rc;
        }
        c->v_valid = false;      // the sweeps below reuse the partials' buffer
        if (c->sym) {
            // V = pre * sum_{i<j} t_ij, every unordered pair evaluated once
            const double pre = c->model == LRMD_RING ? -1.0 / (std::sqrt(2.0) * (double)c->N) : 1.0 / (double)c->N;
            for (const int4& bt : c->sym_batches) {
                SymPart S = c->spart;
                S.tile0 = bt.x; S.tile1 = bt.y; S.w0 = bt.z; S.G = bt.w;
                const dim3 g((unsigned)((S.G + kSymThreads / 32 - 1) / (kSymThreads / 32))), b(kSymThreads);
                if (c->model == LRMD_RING) {
                    if (c->sym_R == 8) L.go(pair_energy_sym_kernel<1, 8>, g, b, (const double2*)js_ptr(c), S, c->eps, pre, vpart(c));
                    else L.go(pair_energy_sym_kernel<1, 4>, g, b, (const double2*)js_ptr(c), S, c->eps, pre, vpart(c));
                } else {
                    if (c->sym_R == 8) L.go(pair_energy_sym_kernel<2, 8>, g, b, (const double2*)js_ptr(c), S, c->eps, pre, vpart(c));
                    else L.go(pair_energy_sym_kernel<2, 4>, g, b, (const double2*)js_ptr(c), S, c->eps, pre, vpart(c));
                }
            }
            L.go(energy_finalize_kernel, dim3(1), dim3(kHmfThreads), c->model, c->N, (const double*)kpart(c), (int)gk,
                 (const double2*)nullptr, 0, (const double*)vpart(c), (int)c->sym_wstart.size(), out4_device);
            return L.rc;
        }
        // V = pre * sum_{i<j} t_ij = (pre/2) * sum_{i != j} t_ij
        with_pair_cfg(c->pair_variant, [&](auto cfg) {
            using CFG = decltype(cfg);
            const dim3 g((unsigned)c->part.G), b(CFG::THREADS);
            if (c->model == LRMD_RING)
                L.go(pair_energy_kernel<1, CFG>, g, b, (const double2*)js_ptr(c), c->part, c->eps,
                     -0.5 / (std::sqrt(2.0) * (double)c->N_total), vpart(c));
            else
                L.go(pair_energy_kernel<2, CFG>, g, b, (const double2*)js_ptr(c), c->part, c->eps, 0.5 / (double)c->N_total,
                     vpart(c));
        });
        L.go(energy_finalize_kernel, dim3(1), dim3(kHmfThreads), c->model, c->N, (const double*)kpart(c), (int)gk,
             (const double2*)nullptr, 0, (const double*)vpart(c), c->part.G, out4_device);
    }
    return L.rc;
}

int lrmd_hmf_forces_static(const double* theta_device, double* f_device, int64_t N, void* cuda_stream,
                           int* cuda_error_host) {
    // no context, no workspace, no allocation: the per-CTA sums go to g_lrmd_static_partials (see above and lrmd.h)
    if (cuda_error_host) *cuda_error_host = 0;
    if (!theta_device || !f_device || N < 1) return LRMD_EINVAL;
    if (((uintptr_t)theta_device % 8) != 0 || ((uintptr_t)f_device % 8) != 0) return LRMD_EINVAL;
    if (N > (int64_t)LRMD_STATIC_MAX_N) return LRMD_ETOOBIG;     // would need more CTA sums than the array holds
    cudaError_t e = cudaSuccess;
    double2* partials = nullptr;
    const int rc = static_partials(&partials, &e);    // first call on this device: looks the address up
    if (rc != LRMD_OK) {
        if (cuda_error_host) *cuda_error_host = (int)e;
        return rc;
    }
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const int ctas = (int)((N + kStaticPerCta - 1) / kStaticPerCta);     // <= kStaticMaxCtas
    long long n = (long long)N;
    const double2* sums = partials;
    {
        void* args[] = {(void*)&theta_device, (void*)&n, (void*)&partials};
        e = cudaLaunchKernel((const void*)hmf_reduce_static_kernel, dim3((unsigned)ctas), dim3(kHmfThreads), args, 0, stream);
    }
    if (e == cudaSuccess) {
        // the force kernel of lrmd_forces, unchanged: every CTA re-sums the `ctas` pairs in index order
        int64_t g = (N + kHmfThreads - 1) / kHmfThreads;
        if (g > kHmfMaxGrid) g = kHmfMaxGrid;
        double inv_n = 1.0 / (double)N;
        int g_in = ctas;
        void* args[] = {(void*)&theta_device, (void*)&f_device, (void*)&n, (void*)&inv_n, (void*)&sums, (void*)&g_in};
        e = cudaLaunchKernel((const void*)hmf_force_kernel, dim3((unsigned)g), dim3(kHmfThreads), args, 0, stream);
    }
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        if (cuda_error_host) *cuda_error_host = (int)e;
        return LRMD_ECUDA;
    }
    return LRMD_OK;
}

int lrmd_set_shard(lrmd_ctx* c, int64_t N_total, int64_t i0, lrmd_allreduce_fn allreduce, lrmd_allgather_fn allgather,
                   void* user) {
    if (!c) return LRMD_EINVAL;
    if (i0 < 0 || N_total < c->N || i0 + c->N > N_total) return LRMD_EINVAL;
    if (c->model != LRMD_HMF && N_total > ((int64_t)1 << 28)) return LRMD_EINVAL;
    const bool shard = N_total != c->N;
    if (shard && (c->model == LRMD_HMF ? !allreduce : !allgather)) return LRMD_EINVAL;
    c->N_total = N_total;
    c->i0 = i0;
    c->allreduce = allreduce;
    c->allgather = allgather;
    c->coll_user = user;
    const Layout before = c->lay;
    const bool had_sym = c->sym;
    resolve(c);
    drop_graph(c);
    c->force_valid = false;
    c->v_valid = false;
    c->js_valid = false;
    rebind_if_changed(c, before, had_sym);
    return LRMD_OK;
}

int lrmd_step_observe(lrmd_ctx* c, int64_t n, double dt, int64_t every, double* out_device, void* cuda_stream) {
    int rc = ready(c);
    if (rc != LRMD_OK) return rc;
    if (n < 0 || every < 1 || !std::isfinite(dt) || !out_device) return LRMD_EINVAL;
    rc = lrmd_energy(c, out_device, cuda_stream);
    int64_t done = 0, rec = 1;
    // band kernel: the force evaluation that ends each lrmd_step call also delivers V (+1 FP64 instruction per pair on
    // one of the 3 evaluations per step instead of a second O(N^2) sweep per record)
    c->want_v = c->band;
    while (rc == LRMD_OK && done + every <= n) {
        rc = lrmd_step(c, every, dt, cuda_stream);
        if (rc == LRMD_OK) rc = lrmd_energy(c, out_device + 4 * rec, cuda_stream);
        done += every;
        ++rec;
    }
    c->want_v = false;
    if (rc == LRMD_OK && done < n) rc = lrmd_step(c, n - done, dt, cuda_stream);
    return rc;
}

int lrmd_set_option(lrmd_ctx* c, int key, int64_t value) {
    if (!c) return LRMD_EINVAL;
    switch (key) {
        case LRMD_OPT_PAIR_PRECISION:
            if (value != 0 && value != 1) return LRMD_EINVAL;
            if (value == 1 && c->model == LRMD_HMF) return LRMD_EUNSUPPORTED;      // fp32 pairs: the pair models
            if (value == 1 && !(c->eps >= 1e-30)) return LRMD_EUNSUPPORTED;        // eps must be a normal float
            c->opt_precision = value;
            break;
        case LRMD_OPT_PAIR_CTAS:
            if (value < 0 || value > (1 << 24)) return LRMD_EINVAL;
            if (c->model == LRMD_HMF && value != 0) return LRMD_EINVAL;
            c->opt_pair_ctas = value;
            break;
        case LRMD_OPT_HMF_VARIANT:
            if (value < -1 || value >= kNumHmfVariants) return LRMD_EINVAL;
            if (c->model != LRMD_HMF && value > 0) return LRMD_EINVAL;
            c->opt_hmf_variant = value;
            break;
        case LRMD_OPT_PAIR_VARIANT:
            if (value < -1 || value >= kNumPairVariants) return LRMD_EINVAL;
            if (c->model == LRMD_HMF && value > 0) return LRMD_EINVAL;
            c->opt_pair_variant = value;
            break;
        case LRMD_OPT_GRAPH:
            if (value < -1 || value > 1) return LRMD_EINVAL;
            c->opt_graph = value;
            break;
        case LRMD_OPT_HMF_GRID:
            if (value < 0 || value > kHmfMaxGrid) return LRMD_EINVAL;
            if (c->model != LRMD_HMF && value != 0) return LRMD_EINVAL;
            c->opt_hmf_grid = value;
            break;
        case LRMD_OPT_PAIR_SYMMETRIC:
            if (value < -1 || value > 2) return LRMD_EINVAL;
            if (c->model == LRMD_HMF && value > 0) return LRMD_EINVAL;
            c->opt_sym = value;
            break;
        case LRMD_OPT_PAIR_FUSE_UPDATE:
            if (value < -1 || value > 1) return LRMD_EINVAL;
            c->opt_fuse = value;
            return LRMD_OK;
        case LRMD_OPT_PAIR_SYM_TILES:
            if (value < 0 || value > (1 << 24)) return LRMD_EINVAL;
            if (c->model == LRMD_HMF && value != 0) return LRMD_EINVAL;
            c->opt_sym_tiles = value;
            break;
        case LRMD_OPT_PAIR_BAND_HEIGHT:
            if (value < 0 || value > (1 << 20)) return LRMD_EINVAL;
            if (c->model == LRMD_HMF && value != 0) return LRMD_EINVAL;
            c->opt_band_height = value;
            break;
        case LRMD_OPT_PAIR_SYM_EXCHANGE:
            if (value < -1 || value > 3) return LRMD_EINVAL;
            if (c->model == LRMD_HMF && value > 0) return LRMD_EINVAL;
            c->opt_sym_xch = value;
            c->sym_xch = value >= 0 ? (int)value : 3;
            return LRMD_OK;
        case LRMD_OPT_KERNEL_TIMING:
            if (value != 0 && value != 1) return LRMD_EINVAL;
            c->timing = value != 0;
            c->ev_used = 0;
            return LRMD_OK;
        default:
            return LRMD_EINVAL;
    }
    const Layout before = c->lay;
    const bool had_sym = c->sym;
    resolve(c);
    drop_graph(c);
    c->force_valid = false;
    c->v_valid = false;
    c->js_valid = false;
    rebind_if_changed(c, before, had_sym);
    return LRMD_OK;
}

int lrmd_get_option(const lrmd_ctx* c, int key, int64_t* value) {
    if (!c || !value) return LRMD_EINVAL;
    switch (key) {
        case LRMD_OPT_PAIR_PRECISION: *value = c->opt_precision; break;
        case LRMD_OPT_PAIR_CTAS: *value = c->model == LRMD_HMF ? 0 : (c->band ? c->bpart.P : (c->sym ? c->spart.G : c->part.G)); break;
        case LRMD_OPT_HMF_VARIANT: *value = c->hmf_variant; break;
        case LRMD_OPT_PAIR_VARIANT: *value = c->pair_variant; break;
        case LRMD_OPT_PAIR_SLOTS: *value = c->band ? (int64_t)c->band_pieces.size() : (c->sym ? c->sym_slots : c->slots); break;
        case LRMD_OPT_PAIR_SYMMETRIC: *value = c->band ? 2 : (c->sym ? 1 : 0); break;
        case LRMD_OPT_PAIR_SYM_TILES: *value = (c->sym && !c->band) ? c->sym_rows : 0; break;
        case LRMD_OPT_PAIR_BAND_HEIGHT: *value = c->band ? c->bpart.hb : 0; break;
        case LRMD_OPT_PAIR_FUSE_UPDATE: *value = ((c->band || (c->sym && c->sym_batches.size() == 1)) && c->opt_fuse != 0) ? 1 : 0; break;
        case LRMD_OPT_GRAPH: *value = c->use_graph ? 1 : 0; break;
        case LRMD_OPT_HMF_GRID: *value = c->hmf_grid; break;
        case LRMD_OPT_KERNEL_TIMING: *value = c->timing ? 1 : 0; break;
        case LRMD_OPT_PAIR_SYM_EXCHANGE:
            if (c->band && c->opt_precision == 1) *value = c->opt_sym_xch <= 0 ? 0 : c->sym_xch;     // fp32 band kernel
            else *value = c->sym ? c->sym_xch : 0;
            break;
        default: return LRMD_EINVAL;
    }
    return LRMD_OK;
}

int lrmd_launch_count(const lrmd_ctx* c, int64_t* launches) {
    if (!c || !launches) return LRMD_EINVAL;
    *launches = c->launches;
    return LRMD_OK;
}

int lrmd_kernel_time(lrmd_ctx* c, double* ms_total_host, int64_t* launches_host) {
    if (!c || !ms_total_host || !launches_host) return LRMD_EINVAL;
    double total = 0.0;
    for (size_t k = 0; k + 1 < c->ev_used; k += 2) {
        cudaError_t e = cudaEventSynchronize(c->ev[k + 1]);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, c->ev[k], c->ev[k + 1]);
        if (e != cudaSuccess) { c->cuda_err = (int)e; (void)cudaGetLastError(); c->ev_used = 0; return LRMD_ECUDA; }
        total += (double)ms;
    }
    *ms_total_host = total;
    *launches_host = (int64_t)(c->ev_used / 2);
    c->ev_used = 0;
    return LRMD_OK;
}

int lrmd_last_cuda_error(const lrmd_ctx* c) { return c ? c->cuda_err : 0; }

const char* lrmd_strerror(int code) {
    switch (code) {
        case LRMD_OK: return "ok";
        case LRMD_EINVAL: return "invalid argument";
        case LRMD_ESTATE: return "state or workspace not set";
        case LRMD_ECUDA: return "CUDA error (see lrmd_last_cuda_error)";
        case LRMD_EUNSUPPORTED: return "not implemented in this build";
        case LRMD_ECOLL: return "a collective callback of a sharded context failed";
        case LRMD_ETOOBIG: return "N exceeds LRMD_STATIC_MAX_N: the library's built-in scratch array is too small, use a context";
        default: return "unknown error code";
    }
}

int lrmd_coefficients(double* out4_host) {
    if (!out4_host) return LRMD_EINVAL;
    const Coef k = coefficients();
    out4_host[0] = k.B0; out4_host[1] = k.B1; out4_host[2] = k.D0; out4_host[3] = k.D1;
    return LRMD_OK;
}

int lrmd_pair_partition(const lrmd_ctx* c, int64_t cta, int64_t* seg4_host, int64_t max_seg, int64_t* nseg_host) {
    if (!c || !nseg_host || c->model == LRMD_HMF || cta < 0 || cta >= c->part.G || max_seg < 0) return LRMD_EINVAL;
    if (max_seg > 0 && !seg4_host) return LRMD_EINVAL;
    int64_t n = 0;
    PairSegments segs(c->part, (long long)cta);
    long long tile, jbeg, jend;
    int slot;
    while (segs.next(c->part, tile, jbeg, jend, slot)) {
        if (n < max_seg) {
            seg4_host[4 * n + 0] = tile;
            seg4_host[4 * n + 1] = jbeg;
            seg4_host[4 * n + 2] = jend;
            seg4_host[4 * n + 3] = slot;
        }
        ++n;
    }
    *nseg_host = n;
    return LRMD_OK;
}

int lrmd_pair_sym_partition(const lrmd_ctx* c, int64_t worker, int64_t* out5_host, int64_t* n_workers_host) {
    if (!c || c->model == LRMD_HMF) return LRMD_EINVAL;
    if (n_workers_host) *n_workers_host = c->sym ? (int64_t)c->sym_wstart.size() : 0;
    if (!out5_host) return n_workers_host ? LRMD_OK : LRMD_EINVAL;
    if (!c->sym || worker < 0 || worker >= (int64_t)c->sym_wstart.size()) return LRMD_EINVAL;
    const int4 st = c->sym_wstart[(size_t)worker];
    int64_t batch = 0;
    for (size_t b = 0; b < c->sym_batches.size(); ++b)
        if (worker >= c->sym_batches[b].z && worker < c->sym_batches[b].z + c->sym_batches[b].w) batch = (int64_t)b;
    out5_host[0] = st.x;                   // first unit: tile
    out5_host[1] = st.y;                   //             chunk of 32 j
    out5_host[2] = st.z;                   // number of (tile, chunk) units, tile-major
    out5_host[3] = batch;                  // launch (batch of tiles) the worker belongs to
    out5_host[4] = 32 * c->sym_R;          // particles per i-tile
    return LRMD_OK;
}

int lrmd_pair_band_partition(const lrmd_ctx* c, int64_t piece, int64_t* out8_host, int64_t* n_pieces_host) {
    if (!c || c->model == LRMD_HMF) return LRMD_EINVAL;
    if (n_pieces_host) *n_pieces_host = c->band ? (int64_t)c->band_pieces.size() : 0;
    if (!out8_host) return n_pieces_host ? LRMD_OK : LRMD_EINVAL;
    if (!c->band || piece < 0 || piece >= (int64_t)c->band_pieces.size()) return LRMD_EINVAL;
    const BandPiece& pc = c->band_pieces[(size_t)piece];
    const BandInfo& bi = c->band_infos[(size_t)pc.band];
    out8_host[0] = pc.band;                          // band of the piece
    out8_host[1] = pc.c0;                            // its columns [c0, c1), in chunks of 32 particles
    out8_host[2] = pc.c1;
    out8_host[3] = c->band_owner[(size_t)piece];     // worker (CTA) that owns it
    out8_host[4] = bi.blk0;                          // the band's I-blocks blk0 .. blk0 + nblk - 1
    out8_host[5] = bi.nblk;
    out8_host[6] = c->bpart.IB;                      // rows per I-block = columns per J-block
    out8_host[7] = c->bpart.P;                       // workers
    return LRMD_OK;
}

int lrmd_fp64_peak(int op, int mix, int extra_per_16, int warps_per_sm, int iters, void* scratch_device,
                   size_t scratch_bytes, double* out4_host, void* cuda_stream) {
    if (!scratch_device || !out4_host || iters < 1 || warps_per_sm < 4 || warps_per_sm > 64 || (warps_per_sm % 4) != 0)
        return LRMD_EINVAL;
    if (((uintptr_t)scratch_device % kAlign) != 0) return LRMD_EINVAL;
    using Kern = void (*)(double*, const double*, int, unsigned long long*);
    Kern kern = nullptr;
#define LRMD_PEAK(OP, XK, XN) if (op == OP && mix == XK && extra_per_16 == XN) kern = fp64_peak_kernel<OP, XK, XN>
    LRMD_PEAK(kPeakDfma, kMixNone, 0); LRMD_PEAK(kPeakDmul, kMixNone, 0); LRMD_PEAK(kPeakDadd, kMixNone, 0);
    LRMD_PEAK(kPeakDfma3, kMixNone, 0); LRMD_PEAK(kPeakDfma2, kMixNone, 0); LRMD_PEAK(kPeakDfmaSq, kMixNone, 0);
    LRMD_PEAK(kPeakDfmaImm, kMixNone, 0);
#define LRMD_PEAK3(XK) LRMD_PEAK(kPeakDfma, XK, 2); LRMD_PEAK(kPeakDfma, XK, 4); LRMD_PEAK(kPeakDfma, XK, 8); LRMD_PEAK(kPeakDfma, XK, 16)
    LRMD_PEAK3(kMixInt); LRMD_PEAK3(kMixMufu); LRMD_PEAK3(kMixShfl); LRMD_PEAK3(kMixLds); LRMD_PEAK3(kMixMufuSeed);
    LRMD_PEAK3(kMixMov); LRMD_PEAK3(kMixSts);
#undef LRMD_PEAK3
#undef LRMD_PEAK
    if (!kern) return LRMD_EUNSUPPORTED;
    const int grid = kNumSm * (warps_per_sm / (kPeakThreads / 32));
    const size_t out_bytes = align_up(sizeof(double) * (size_t)grid * kPeakThreads);
    const size_t seed_bytes = align_up(sizeof(double) * 4);
    const size_t clk_bytes = align_up(sizeof(unsigned long long) * 2 * (size_t)grid);
    if (scratch_bytes < out_bytes + seed_bytes + clk_bytes) return LRMD_EINVAL;
    char* base = static_cast<char*>(scratch_device);
    double* out = reinterpret_cast<double*>(base);
    double* seedv = reinterpret_cast<double*>(base + out_bytes);
    unsigned long long* clk = reinterpret_cast<unsigned long long*>(base + out_bytes + seed_bytes);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    // operands of the chains: a <- a * m + c stays finite and normal for any number of iterations
    const double seed[4] = {0.99999999, 1.0e-3, 1.0, 0.0};
    std::vector<unsigned long long> hclk(2 * (size_t)grid);
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    cudaError_t e = cudaMemcpyAsync(seedv, seed, sizeof(seed), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    float ms = 0.f;
    if (e == cudaSuccess) {
        kern<<<grid, kPeakThreads, 0, st>>>(out, seedv, iters > 64 ? 64 : iters, clk);     // warm-up
        cudaEventRecord(e0, st);
        kern<<<grid, kPeakThreads, 0, st>>>(out, seedv, iters, clk);
        cudaEventRecord(e1, st);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaEventSynchronize(e1);
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    if (e == cudaSuccess) e = cudaMemcpyAsync(hclk.data(), clk, sizeof(unsigned long long) * hclk.size(), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return LRMD_ECUDA; }
    double cyc = 0.0, ns = 0.0;
    for (int b = 0; b < grid; ++b) { cyc += (double)hclk[2 * b]; ns += (double)hclk[2 * b + 1]; }
    const double fp64_per_thread = (double)iters * (kPeakChains + (mix == kMixMufuSeed ? extra_per_16 : 0));
    const double instr = fp64_per_thread * (double)grid * kPeakThreads;     // thread-level FP64 instructions
    const double mhz = ns > 0.0 ? cyc / ns * 1e3 : 0.0;
    out4_host[0] = instr / ((double)ms * 1e-3);                               // FP64 instructions per second
    out4_host[1] = mhz;                                                       // SM clock held (clock64 / globaltimer)
    out4_host[2] = mhz > 0.0 ? out4_host[0] / (mhz * 1e6 * kNumSm) : 0.0;    // FP64 lanes busy per clock per SM
    out4_host[3] = (double)ms;
    return LRMD_OK;
}

int lrmd_host_sincos(const double* x_host, int64_t n, double* s_host, double* c_host) {
    if (!x_host || !s_host || !c_host || n < 0) return LRMD_EINVAL;
    for (int64_t i = 0; i < n; ++i) sincos_any(x_host[i], s_host[i], c_host[i]);
    return LRMD_OK;
}

}  // extern "C"
