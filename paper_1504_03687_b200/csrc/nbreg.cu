// nbreg.cu -- host side of libnbreg: context, launch planning, the extern "C" entry points of
// include/nbreg.h.  No torch types, no CPU fallback: every step of the path runs in the kernels of
// nbreg_kernels.cuh on an sm_100 device or the call fails.
#include "../../include/nbreg.h"
#include "nbreg_kernels.cuh"

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <unordered_map>

using namespace nbreg;

namespace {

struct Variant {
    int it, wi, wj;          // i per thread, warps along i, warps along j
    int iblock;              // i-particles per CTA
    int threads;
    size_t smem;             // dynamic shared memory of one CTA (ForceSmem<...>::TOTAL)
    double ovh_tiles;        // per-CTA fixed cost in units of one tile's compute (planning heuristic)
    int ctas_per_sm;         // from the occupancy API at nb_open
};
constexpr int NVARIANT = 5;
constexpr int NAUTO = 5;        // variants the planner picks from; the rest only by NB_TUNE_FORCE_VARIANT
constexpr int FUSED_FIRST = 2;  // variants 2..4 (128, 64, 32 i per CTA) also exist reading the FP64 state (fused predictor)
constexpr double DEFAULT_LOCAL_G = 8.0;     // local-frame guard |x_i - c| <= G h_i

}  // namespace

struct nb_ctx {
    int64_t N = 0, Npad = 0, Ns = 0;
    int32_t cap = 0;
    int sm_count = 0;
    int device = 0;                         // the CUDA device the context lives on
    double pred_t = 0.0;                    // time of the last nb_predict_all / nb_step_host (valid when have_pred)
    cudaStream_t stream = nullptr;
    cudaError_t cuda_err = cudaSuccess;
    bool have_j = false, have_pred = false;
    bool pred_pending = false;              // nb_predict_all(t) was called but the records are not written yet:
                                            // a small block predicts inside the force kernel instead (fused path)
    bool fuse = true;                       // NB_TUNE_FUSE_PREDICT
    double local_g = DEFAULT_LOCAL_G;       // NB_TUNE_LOCAL_G_MILLI / 1000
    unsigned int *stats = nullptr;          // {warps in the local frame, warps} since NB_TUNE_STATS was set
    // Morton reordering of large blocks (reorder_block): sort scratch, bounding box
    int64_t reorder_min = 4096;             // NB_TUNE_REORDER_MIN: blocks of at least this many particles; 0 = never
    unsigned long long *sort_keys = nullptr;   // after the sort: slot -> k = key & PERM_MASK
    uint32_t *sort_box = nullptr;
    int64_t sort_n = 0;
    int64_t last_reordered = 0;
    // device state owned by the library
    double *soa = nullptr;                  // [14][Ns]
    double *aos = nullptr;                  // [N][16] gather copy (one 128 B line per body); allocated and built by the
                                            // first NEXT-2 / NEXT-3 call (ensure_aos), kept current from then on
    int sort_P = 0; size_t sort_smem_max = 0;   // list-row sort: power of two >= cap; opt-in dynamic smem limit
    float *rec = nullptr;                   // predicted records [Npad / TJ][RECF][TJ]
    int32_t *cnt = nullptr;                 // [cnt_n >= N] zero between calls
    int64_t cnt_n = 0;
    double *partial = nullptr;  size_t partial_bytes = 0;
    // staging for the HOST variants (lazy)
    double *stage_j = nullptr;              // 14 N doubles
    int32_t *st_idx = nullptr, *st_nnb = nullptr, *st_ovf = nullptr, *st_list = nullptr;
    double *st_h2 = nullptr, *st_out = nullptr;     // st_out: acc[3n] jerk[3n] pot[n]
    int64_t st_n = 0, st_list_n = 0;
    // pipelined HOST step (nb_step_host): copy stream, per-chunk events, the active particles' own state
    static constexpr int MAXCHUNK = 8;
    cudaStream_t copy_stream = nullptr, prep_stream = nullptr;   // H2D copies / re-layout + predictor of landed chunks
    cudaStream_t force_stream[MAXCHUNK] = {};                    // one per chunk: the per-chunk force launches overlap
    cudaEvent_t ev_force[MAXCHUNK] = {}, ev_iready = nullptr;
    cudaEvent_t ev_enter = nullptr, ev_i = nullptr, ev_copied[MAXCHUNK] = {}, ev_chunk[MAXCHUNK] = {};
    double *h_ist = nullptr, *d_ist = nullptr;      // [14][n_i] gathered FP64 state (pinned host / device)
    float *irec = nullptr;                          // [RECF][n_i_pad] their predicted records
    int64_t ist_n = 0;
    // block loop (NEXT-3): steps, selection scratch
    double *dtj = nullptr;                          // [N] block time steps
    bool have_steps = false;
    unsigned long long *sel_key = nullptr;          // min_j (t0 + dt) as an ordered integer key
    int32_t *sel_counts = nullptr;                  // [ceil(N / SEL_CHUNK)]
    double *sel_result = nullptr, *h_sel_result = nullptr;   // {t_next, n_active}: device / pinned host
    // nb_block_step: one cooperative selection launch (two alternating minimum slots), the block's own buffers
    unsigned long long *blk_key = nullptr;          // [2]
    int blk_parity = 0;
    int32_t *blk_idx = nullptr;                     // [N] active indices of the last block
    double *blk_out = nullptr;                      // acc[3n] jerk[3n] pot[n]
    int32_t *blk_nnb = nullptr, *blk_ovf = nullptr, *blk_list = nullptr;
    int64_t blk_n = 0, blk_list_n = 0, blk_last_n = 0;
    bool blk_had_list = false;
    int32_t ac_fail_nr = 0;                         // regular rows of the two-level block that returned NB_EOVERFLOW (0: none)
    bool blk_last_two = false;                      // the last block loop was the two-level one (nb_get_block: NB_ESTATE)
    int32_t h2_by_body = 0;                         // the h2 array of the launch in flight is indexed by body
    const double *spec_dev = nullptr;               // non-NULL while a SPECULATIVE chain is enqueued: the kernels take the
                                                    // block's {t, n, status} from this device address
    int64_t blk_stride = 0;                         // acc / jerk / pot of the last block sit at 0, 3, 6 x this in blk_out
    // two-level AC stepping (nb_ac_init / nb_ac_step): per-body force polynomials, persistent lists, scratch
    AcState ac = {};
    double *ac_h2 = nullptr, *ac_aIo = nullptr, *ac_jIo = nullptr;     // radii; irregular force over the old list (by body)
    int32_t *ac_reg_idx = nullptr, *ac_novf = nullptr, *h_ac_novf = nullptr;
    double *ac_in = nullptr;                                           // new-list irregular force of a block: acc[3n] jerk[3n]
    int64_t ac_in_n = 0;
    bool have_ac = false;
    double *blk_ring = nullptr, *h_blk_ring = nullptr;                 // descriptors of a batch of blocks: {t, n, n_reg, status}
    unsigned long long *blk_pub = nullptr;                             // per-chunk counts of the selection, epoch-tagged
    uint32_t blk_epoch = 0;
    unsigned long long *sel_cmin = nullptr;                            // [chunks of SEL_CHUNK bodies] min of t0 + dt, kept between blocks
    int32_t *sel_dirty = nullptr;                                      // [chunks] set by the correctors: rescan this chunk
    bool sel_all_dirty = true;                                         // the state or the steps were replaced: rescan everything
    bool sel_chunks = true;                                            // NB_TUNE_SELECT_CHUNKS
    int64_t sel_grid_max = 0;          // CTAs of select_scatter_kernel the device holds at once (blk_setup)
    int64_t sel_grid_cap = 0;          // NB_TUNE_SELECT_GRID: a smaller cap (0 = none)
    double *p64 = nullptr;                                             // [N][8] FP64 predicted records of a large block's neighbour force
    int64_t irr_pred_min = 49152;                                      // NB_TUNE_IRR_PRED_MIN: blocks of at least this many bodies use them
    int32_t *blk_stall = nullptr;                                      // set by the first block of a batch that needs the host
    bool blk_stall_dirty = true;                                       // the flag must be cleared before the next batch
    int blk_batch = 1;                                                 // blocks enqueued per host round trip (adaptive)
    int64_t spec_hits = 0, spec_misses = 0, blk_prev_n = 0;
    bool spec_enabled = true;                       // NB_TUNE_SPECULATE
    // planning / introspection
    Variant var[NVARIANT];                  // reading the predicted records
    Variant fvar[NVARIANT];                 // reading the FP64 state (entries FUSED_FIRST.. only)
    int64_t last_fused = 0;
    int64_t launches = 0;
    int64_t last_S = 0, last_iblock = 0, last_grid = 0, last_variant = -1;
    int64_t force_S = 0, force_variant = -1, step_chunks = 0;
    int64_t j_offset = 0;                           // global index of body 0 (j-sharding)
    std::unordered_map<int64_t, int> plan_cache;   // (j-tiles, variant, i-blocks) -> S
    // optional event bracketing of the force kernel (NB_TUNE_PROFILE)
    static constexpr int PROF_RING = 256;
    bool profile = false;
    cudaEvent_t ev0[PROF_RING] = {}, ev1[PROF_RING] = {};
    int64_t prof_n = 0;
};

namespace {

#define NB_CUDA(ctx, expr)                          \
    do {                                            \
        cudaError_t e__ = (expr);                   \
        if (e__ != cudaSuccess) {                   \
            (ctx)->cuda_err = e__;                  \
            return e__ == cudaErrorMemoryAllocation ? NB_ENOMEM : NB_ECUDA; \
        }                                           \
    } while (0)

template <int WI, int WJ, int MINB, bool JP = false, int SRC = SRC_REC>
cudaError_t setup_variant(Variant &v, double ovh) {
    v.it = JP ? 1 : 2; v.wi = WI; v.wj = WJ; v.iblock = (JP ? 32 : 64) * WI; v.threads = 32 * WI * WJ; v.ovh_tiles = ovh;
    v.smem = ForceSmem<WI, WJ, JP, SRC>::TOTAL;
    auto k = force_kernel<WI, WJ, MINB, JP, SRC>;
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)v.smem);
    if (e != cudaSuccess) return e;
    int nb = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, k, v.threads, v.smem);
    v.ctas_per_sm = std::max(nb, 1);
    return e;
}

// Launch with programmatic stream serialization: the grid is placed while its predecessor in the stream drains, so
// the launch latency is not on the path of a chain of short kernels (block loop; nb_regular of a small block).  Every
// kernel launched this way starts with pdl_wait() (griddepcontrol.wait) before it reads anything.
template <typename... KArgs, typename... Args>
cudaError_t launch_chain(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args &&...args) {
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(std::forward<Args>(args))...);
}

template <int WI, int WJ, int MINB, bool JP = false, int SRC = SRC_REC>
void launch_force(const Variant &v, dim3 grid, cudaStream_t st, const ForceParams &p) {
    launch_chain(force_kernel<WI, WJ, MINB, JP, SRC>, grid, dim3(v.threads), v.smem, st, p);
}

// i-particles per CTA, planning overhead (in tile units) and relative cost per padded i-slot of the
// variants <8,1>, <4,2>, <2,4>, <1,8> and the j-packed <1,8> (32 i per CTA).  The cost factors are
// measured: time per padded i-slot at n_i = 8256 and 16500, N = 1M, relative to <8,1>.
constexpr int VAR_IBLOCK[NVARIANT] = {512, 256, 128, 64, 32};
// Planning model, fitted to launches of n_i = 4096 .. 16384 at N = 1M with 19 .. 148 splits (B200):
//   time ~ (waves + TAIL) x (tiles per split + per-CTA overhead) + finalize cost per split
// in units of one tile's compute of the variant.  A CTA's tile takes iblock x 256 pairs at half an SM's rate
// (two CTAs share it: 3.6e9 pairs/s), its prologue + epilogue about 5 us, and the final reduction reads one
// more partial row per split (~0.005 us each).  TAIL: the last wave drains with half-empty SMs.
constexpr double PLAN_TAIL = 0.13, PLAN_CTA_US = 5.0, PLAN_FIN_US_PER_SPLIT = 0.005;
constexpr double var_tile_us(int v) { return VAR_IBLOCK[v] * 256.0 / 3.6e9 * 1.0e6; }
constexpr double VAR_OVH[NVARIANT] = {PLAN_CTA_US / var_tile_us(0), PLAN_CTA_US / var_tile_us(1), PLAN_CTA_US / var_tile_us(2),
                                      PLAN_CTA_US / var_tile_us(3), PLAN_CTA_US / var_tile_us(4)};
constexpr double VAR_COST[NVARIANT] = {1.0, 1.01, 1.025, 1.03, 1.11};

// Pick the kernel variant: least padded work weighted by the variant's rate, ties to the larger i-block
// (more reuse of each j load).
int pick_variant_pure(int64_t n_i) {
    int best = 0;
    double best_cost = -1.0;
    for (int v = 0; v < NAUTO; ++v) {
        const int64_t ib = VAR_IBLOCK[v];
        const double cost = (double)((n_i + ib - 1) / ib * ib) * VAR_COST[v];
        if (best_cost < 0.0 || cost < best_cost) { best = v; best_cost = cost; }
    }
    return best;
}
int pick_variant(const nb_ctx *c, int32_t n_i) {
    if (c->force_variant >= 0 && c->force_variant < NVARIANT) return (int)c->force_variant;
    return pick_variant_pure(n_i);
}
// Pick the number of j-splits S: minimise waves x (tiles per split + per-CTA overhead); among plans
// within 0.3 % take the smallest S (less scratch, shorter final reduction).
int plan_split(const nb_ctx *c, const Variant &v, int64_t n_ib, int64_t ntiles);
int plan_split_pure(int64_t conc, double ovh_tiles, double tile_us, int64_t n_ib, int64_t ntiles);
int plan_chunks_pure(int64_t ntiles, int64_t want, int64_t *ctile);

int pick_split(nb_ctx *c, const Variant &v, int64_t n_ib, int64_t ntiles) {
    if (c->force_S > 0) return (int)std::min<int64_t>(c->force_S, ntiles);
    const bool fused = &v >= c->fvar && &v < c->fvar + NVARIANT;
    const int64_t key = (ntiles << 32) ^ (n_ib * 2 * NVARIANT + (fused ? NVARIANT + (&v - c->fvar) : (&v - c->var)));
    auto hit = c->plan_cache.find(key);
    if (hit != c->plan_cache.end()) return hit->second;
    const int plan = plan_split(c, v, n_ib, ntiles);
    c->plan_cache.emplace(key, plan);
    return plan;
}

int plan_split(const nb_ctx *c, const Variant &v, int64_t n_ib, int64_t ntiles) {
    return plan_split_pure((int64_t)c->sm_count * v.ctas_per_sm, v.ovh_tiles, v.iblock * 256.0 / 3.6e9 * 1.0e6, n_ib, ntiles);
}

int plan_split_pure(int64_t conc, double ovh_tiles, double tile_us, int64_t n_ib, int64_t ntiles) {
    const int64_t smax = std::min<int64_t>(ntiles, 8192);
    auto cost = [&](int64_t S, int64_t &Seff) {
        const int64_t tps = (ntiles + S - 1) / S;
        Seff = (ntiles + tps - 1) / tps;                     // splits that actually get tiles
        const int64_t waves = (n_ib * Seff + conc - 1) / conc;
        return ((double)waves + PLAN_TAIL) * ((double)tps + ovh_tiles) + PLAN_FIN_US_PER_SPLIT * (double)Seff / tile_us;
    };
    double best = 1e300;
    int64_t Seff = 1;
    for (int64_t S = 1; S <= smax; ++S) best = std::min(best, cost(S, Seff));
    for (int64_t S = 1; S <= smax; ++S)
        if (cost(S, Seff) <= best * 1.015) return (int)Seff;      // within the model's accuracy: fewer splits, less scratch
    return 1;
}

// Chunk plan of nb_step_host: tile boundaries ctile[0..nchunk] of chunks sized 1/2^L, 1/2^L, then
// doubling (L = 4: 1/16, 1/16, 1/8, 1/4, 1/2), so that the first copy is short and every later copy hides
// behind the force launches of the chunks before it.  want = 0: automatic L from the problem size.
int plan_chunks_pure(int64_t ntiles, int64_t want, int64_t *ctile) {
    constexpr int MAXCHUNK = 8;
    int L = ntiles >= 2048 ? 4 : ntiles >= 512 ? 2 : 0;
    if (want > 0) L = (int)std::min<int64_t>(want - 1, MAXCHUNK - 1);
    while (L > 0 && (ntiles >> L) == 0) --L;
    int64_t sz = std::max<int64_t>(ntiles >> L, 1), at = 0;
    int nchunk = 0;
    ctile[0] = 0;
    while (at < ntiles) {
        const bool last = (nchunk == L) || (at + sz >= ntiles);
        at = last ? ntiles : at + sz;
        ctile[++nchunk] = at;
        if (nchunk >= 2) sz *= 2;
    }
    return nchunk;
}

int check_live(nb_ctx *c) {
    if (!c) return NB_EINVAL;
    if (c->cuda_err != cudaSuccess) return NB_ECUDA;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != c->device) return NB_ESTATE;   // called with another device current
    return NB_OK;
}

int ensure_partial(nb_ctx *c, size_t bytes) {
    if (bytes <= c->partial_bytes) return NB_OK;
    if (c->partial) {
        NB_CUDA(c, cudaStreamSynchronize(c->stream));
        NB_CUDA(c, cudaFree(c->partial));
        c->partial = nullptr; c->partial_bytes = 0;
    }
    const size_t want = bytes + bytes / 4;
    NB_CUDA(c, cudaMalloc(&c->partial, want));
    c->partial_bytes = want;
    return NB_OK;
}

// One force-kernel launch over the j-tiles [tile0, tile1) split S ways, writing partial rows
// [split0, split0 + S).
int launch_force_range(nb_ctx *c, int vi, bool fused, int32_t n_i, const int32_t *idx_i, const double *h2_i,
                       const float *irec, const unsigned long long *perm, int64_t j_offset, int32_t *nblist, int64_t tile0,
                       int64_t tile1, int S, int64_t split0, cudaStream_t st = nullptr, bool own_stream = true) {
    if (own_stream) st = c->stream;
    const Variant &v = fused ? c->fvar[vi] : c->var[vi];
    const int64_t n_ib = (n_i + v.iblock - 1) / v.iblock;
    ForceParams p;
    p.rec = c->rec;
    p.soa = c->soa; p.Ns = c->Ns; p.t = c->pred_t;
    p.g2 = (float)(c->local_g * c->local_g); p.stats = c->stats;
    p.blk_dev = c->spec_dev;
    p.idx_i = idx_i; p.h2_i = h2_i; p.perm = perm; p.h2_by_body = c->h2_by_body;
    p.n_i = n_i; p.n_i_pad = (int32_t)(n_ib * v.iblock);
    p.irec = irec;
    p.tile0 = (int32_t)tile0; p.ntiles = (int32_t)tile1; p.split0 = (int32_t)split0;
    p.j_offset = (int32_t)j_offset;     // 0 except from nb_regular_shard (idx_i global there)
    p.tiles_per_split = (int32_t)((tile1 - tile0 + S - 1) / S);
    p.cap = c->cap; p.cnt = c->cnt; p.nblist = nblist; p.partial = c->partial;
    const dim3 grid((unsigned)n_ib, (unsigned)S);
    const int slot = (int)(c->prof_n % nb_ctx::PROF_RING);
    if (c->profile) NB_CUDA(c, cudaEventRecord(c->ev0[slot], st));
    if (fused) {
        switch (vi) {
            case 2: launch_force<2, 4, 2, false, SRC_STATE>(v, grid, st, p); break;
            case 3: launch_force<1, 8, 2, false, SRC_STATE>(v, grid, st, p); break;
            default: launch_force<1, 8, 2, true, SRC_STATE>(v, grid, st, p); break;
        }
    } else {
        switch (vi) {
            case 0: launch_force<8, 1, 2>(v, grid, st, p); break;
            case 1: launch_force<4, 2, 2>(v, grid, st, p); break;
            case 2: launch_force<2, 4, 2>(v, grid, st, p); break;
            case 3: launch_force<1, 8, 2>(v, grid, st, p); break;
            default: launch_force<1, 8, 2, true>(v, grid, st, p); break;
        }
    }
    NB_CUDA(c, cudaGetLastError());
    if (c->profile) {
        NB_CUDA(c, cudaEventRecord(c->ev1[slot], st));
        c->prof_n += 1;
    }
    c->launches += 1;
    c->last_iblock = v.iblock; c->last_grid = n_ib * S; c->last_variant = vi; c->last_fused = fused ? 1 : 0;
    return NB_OK;
}

// nb_predict_all defers the predictor launch (pred_pending); whoever needs the records calls this first.
int materialize_pred(nb_ctx *c) {
    if (!c->pred_pending) return NB_OK;
    predict_kernel<<<(unsigned)((c->Npad + 255) / 256), 256, 0, c->stream>>>(0, c->Npad, c->N, c->Ns, c->pred_t, c->soa, c->rec);
    NB_CUDA(c, cudaGetLastError());
    c->launches += 1;
    c->pred_pending = false;
    return NB_OK;
}

// The 128 B/body gather copy of the state (NEXT-2 / NEXT-3 kernels): built on first use.
int ensure_aos(nb_ctx *c) {
    if (c->aos) return NB_OK;
    NB_CUDA(c, cudaMalloc(&c->aos, sizeof(double) * AOS_D * c->N));
    soa_to_aos_kernel<<<(unsigned)((c->N + 255) / 256), 256, 0, c->stream>>>(c->N, c->Ns, c->soa, c->aos);
    NB_CUDA(c, cudaGetLastError());
    c->launches += 1;
    return NB_OK;
}

// NEXT-2 launch: the neighbour force of n bodies at time t.  A large block (not a speculative launch, whose size
// the host does not know) predicts every body once into 64 B records and gathers those (irregular_kernel<., true>);
// p64_ready: the records of this t are in place already (second pass of the same block).
template <bool ACCUM>
int launch_irregular(nb_ctx *c, bool chain, int32_t n, double t, const double *dev, int32_t rows_by_body, int32_t out_by_body,
                     const int32_t *idx, const int32_t *nnb, const int32_t *list, double *acc, double *jerk, double *pot,
                     bool p64_ready = false) {
    const bool pred = dev == nullptr && c->irr_pred_min > 0 && n >= c->irr_pred_min;
    if (pred && !p64_ready) {
        if (!c->p64) NB_CUDA(c, cudaMalloc(&c->p64, sizeof(double) * P64_D * c->N));
        predict64_kernel<<<(unsigned)((c->N + 255) / 256), 256, 0, c->stream>>>(c->N, t, c->aos, c->p64);
        NB_CUDA(c, cudaGetLastError());
        c->launches += 1;
    }
    const dim3 grid((unsigned)((n + 7) / 8)), block(256);
    const double *src = pred ? c->p64 : c->aos;
    if (chain) {
        if (pred) NB_CUDA(c, launch_chain(irregular_kernel<ACCUM, true>, grid, block, 0, c->stream, n, c->cap, t, dev, rows_by_body,
                                          out_by_body, idx, nnb, list, src, acc, jerk, pot));
        else NB_CUDA(c, launch_chain(irregular_kernel<ACCUM, false>, grid, block, 0, c->stream, n, c->cap, t, dev, rows_by_body,
                                     out_by_body, idx, nnb, list, src, acc, jerk, pot));
    } else {
        if (pred) irregular_kernel<ACCUM, true><<<grid, block, 0, c->stream>>>(n, c->cap, t, dev, rows_by_body, out_by_body, idx, nnb,
                                                                              list, src, acc, jerk, pot);
        else irregular_kernel<ACCUM, false><<<grid, block, 0, c->stream>>>(n, c->cap, t, dev, rows_by_body, out_by_body, idx, nnb,
                                                                          list, src, acc, jerk, pot);
        NB_CUDA(c, cudaGetLastError());
    }
    c->launches += 1;
    return NB_OK;
}

// a6-a7: fixed-order sum of the S partial rows, counters, sorted list rows.  perm (or NULL): slot -> k of
// a block the library reordered (Morton order, reorder_block).
int launch_finalize(nb_ctx *c, int32_t n_i, int64_t n_i_pad, int S, const unsigned long long *perm, double *acc, double *jerk,
                    double *pot, int32_t *nnb, int32_t *nblist, int32_t *overflow) {
    // small blocks: 16 warps share the S partial rows (latency); large blocks have CTAs enough: 4 warps, and a
    // row's sort gets a 128-thread CTA
    const int W = (S > 8 && n_i <= 512) ? 16 : 4;
    const size_t row_bytes = (size_t)c->sort_P * sizeof(int32_t);
    const int sortP = (nblist && row_bytes <= c->sort_smem_max) ? c->sort_P : 0;   // 0: rows stay in append order
    const dim3 fgrid((unsigned)((n_i + 31) / 32), (unsigned)(7 + 32));
    const size_t smem = sortP ? row_bytes : 0;
    // Programmatic dependent launch: the finalize grid is placed while the force kernel drains and
    // waits (griddepcontrol.wait) for its completion, so the launch latency is not on the path of
    // small blocks.
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = fgrid;
    cfg.blockDim = dim3(W == 4 ? 128 : 512);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = c->stream;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    const int32_t n_i_pad32 = (int32_t)n_i_pad, S32 = S, cap32 = c->cap, sortP32 = sortP;
    const double *partial = c->partial, *blk_dev = c->spec_dev;
    if (W == 4)
        NB_CUDA(c, cudaLaunchKernelEx(&cfg, finalize_kernel<4>, n_i, n_i_pad32, S32, cap32, sortP32, perm, blk_dev,
                                      partial, c->cnt, acc, jerk, pot, nnb, nblist, overflow));
    else
        NB_CUDA(c, cudaLaunchKernelEx(&cfg, finalize_kernel<16>, n_i, n_i_pad32, S32, cap32, sortP32, perm, blk_dev,
                                      partial, c->cnt, acc, jerk, pot, nnb, nblist, overflow));
    NB_CUDA(c, cudaGetLastError());
    c->launches += 1;
    c->last_S = S;
    return NB_OK;
}

// Morton order of a large block (a3): c->sort_keys[slot] & PERM_MASK = k afterwards.  Reads the predicted
// records of the active particles (irec if given, else rec[idx_i[k]]); everything on the context's stream.
int reorder_block(nb_ctx *c, int32_t n_i, const int32_t *idx_i, const float *irec, int64_t n_i_pad) {
    int64_t n2 = 2;
    while (n2 < n_i) n2 <<= 1;
    if (n2 > c->sort_n) {
        NB_CUDA(c, cudaStreamSynchronize(c->stream));
        cudaFree(c->sort_keys);
        c->sort_keys = nullptr; c->sort_n = 0;
        NB_CUDA(c, cudaMalloc(&c->sort_keys, sizeof(unsigned long long) * n2));
        c->sort_n = n2;
    }
    if (!c->sort_box) NB_CUDA(c, cudaMalloc(&c->sort_box, 6 * sizeof(uint32_t)));
    NB_CUDA(c, cudaMemsetAsync(c->sort_box, 0xff, 6 * sizeof(uint32_t), c->stream));
    const unsigned gb = (unsigned)std::min<int64_t>((n_i + 255) / 256, (int64_t)c->sm_count * 4);
    block_bbox_kernel<<<gb, 256, 0, c->stream>>>(n_i, n_i_pad, idx_i, c->rec, irec, c->sort_box);
    morton_key_kernel<<<(unsigned)((n2 + 255) / 256), 256, 0, c->stream>>>(n_i, (int32_t)n2, n_i_pad, idx_i, c->rec, irec,
                                                                          c->sort_box, c->sort_keys);
    const int64_t ch = std::min<int64_t>(n2, SORT_CH);
    const unsigned chunks = (unsigned)(n2 / ch);
    bitonic_chunk_kernel<0><<<chunks, SORT_T, 0, c->stream>>>((int32_t)n2, 0, c->sort_keys);
    c->launches += 3;
    for (int64_t size = 2 * ch; size <= n2; size <<= 1) {
        for (int64_t stride = size / 2; stride >= ch; stride >>= 1) {
            bitonic_global_kernel<<<(unsigned)((n2 / 2 + 255) / 256), 256, 0, c->stream>>>((int32_t)n2, (int32_t)size,
                                                                                          (int32_t)stride, c->sort_keys);
            c->launches += 1;
        }
        bitonic_chunk_kernel<1><<<chunks, SORT_T, 0, c->stream>>>((int32_t)n2, (int32_t)size, c->sort_keys);
        c->launches += 1;
    }
    NB_CUDA(c, cudaGetLastError());
    return NB_OK;
}
bool want_reorder(const nb_ctx *c, int32_t n_i) {
    return c->local_g > 0.0 && c->reorder_min > 0 && n_i >= c->reorder_min && (int64_t)n_i <= (int64_t)PERM_MASK;
}

int regular_device(nb_ctx *c, int32_t n_i, const int32_t *idx_i, const double *h2_i, double *acc, double *jerk,
                   double *pot, int32_t *nnb, int32_t *nblist, int32_t *overflow) {
    const int vi = pick_variant(c, n_i);
    const int64_t n_ib = (n_i + c->var[vi].iblock - 1) / c->var[vi].iblock;
    // Small blocks (one i-block: every j-tile has exactly one reader) whose prediction is still pending
    // read the FP64 state and predict inside the force kernel; everything else needs the records.
    const bool fused = c->pred_pending && c->fuse && vi >= FUSED_FIRST && n_ib == 1;
    // A speculative chain knows its block time only on the device: only the fused kernel reads it from there.  The
    // records route would predict all N bodies to the host's placeholder time (run_blocks never asks for this).
    if (c->spec_dev && !fused) return NB_ESTATE;
    int rc = fused ? NB_OK : materialize_pred(c);
    if (rc != NB_OK) return rc;
    const Variant &v = fused ? c->fvar[vi] : c->var[vi];
    const int64_t ntiles = c->Npad / TJ;
    const int S = pick_split(c, v, n_ib, ntiles);
    const int64_t n_i_pad = n_ib * v.iblock;
    rc = ensure_partial(c, (size_t)S * 7 * n_i_pad * sizeof(double));
    if (rc != NB_OK) return rc;
    const unsigned long long *perm = nullptr;
    c->last_reordered = 0;
    if (!fused && want_reorder(c, n_i)) {
        rc = reorder_block(c, n_i, idx_i, nullptr, n_i_pad);
        if (rc != NB_OK) return rc;
        perm = c->sort_keys; c->last_reordered = 1;
    }
    rc = launch_force_range(c, vi, fused, n_i, idx_i, h2_i, nullptr, perm, 0, nblist, 0, ntiles, S, 0);
    if (rc != NB_OK) return rc;
    return launch_finalize(c, n_i, n_i_pad, S, perm, acc, jerk, pot, nnb, nblist, overflow);
}

// Device-side buffers of the HOST variants, grown on demand.
int ensure_host_staging(nb_ctx *c, int32_t n_i, bool want_list) {
    if (n_i > c->st_n) {
        NB_CUDA(c, cudaStreamSynchronize(c->stream));
        cudaFree(c->st_idx); cudaFree(c->st_nnb); cudaFree(c->st_ovf); cudaFree(c->st_h2); cudaFree(c->st_out);
        c->st_idx = c->st_nnb = c->st_ovf = nullptr; c->st_h2 = c->st_out = nullptr; c->st_n = 0;
        const int64_t n = std::min<int64_t>(c->N, std::max<int64_t>(n_i, 1024) * 5 / 4);
        NB_CUDA(c, cudaMalloc(&c->st_idx, sizeof(int32_t) * n));
        NB_CUDA(c, cudaMalloc(&c->st_nnb, sizeof(int32_t) * n));
        NB_CUDA(c, cudaMalloc(&c->st_ovf, sizeof(int32_t) * n));
        NB_CUDA(c, cudaMalloc(&c->st_h2, sizeof(double) * n));
        NB_CUDA(c, cudaMalloc(&c->st_out, sizeof(double) * 7 * n));
        c->st_n = n;
    }
    const int64_t need_list = want_list ? (int64_t)n_i * c->cap : 0;
    if (need_list > c->st_list_n) {
        NB_CUDA(c, cudaStreamSynchronize(c->stream));
        cudaFree(c->st_list); c->st_list = nullptr; c->st_list_n = 0;
        NB_CUDA(c, cudaMalloc(&c->st_list, sizeof(int32_t) * need_list));
        c->st_list_n = need_list;
    }
    return NB_OK;
}

// Copy the staged outputs of a HOST variant back and wait for them.
int copy_back(nb_ctx *c, int32_t n_i, double *acc, double *jerk, double *pot, int32_t *nnb, int32_t *nblist,
              int32_t *overflow) {
    const double *d_acc = c->st_out, *d_jerk = c->st_out + 3 * (int64_t)n_i, *d_pot = c->st_out + 6 * (int64_t)n_i;
    NB_CUDA(c, cudaMemcpyAsync(acc, d_acc, sizeof(double) * 3 * n_i, cudaMemcpyDeviceToHost, c->stream));
    NB_CUDA(c, cudaMemcpyAsync(jerk, d_jerk, sizeof(double) * 3 * n_i, cudaMemcpyDeviceToHost, c->stream));
    NB_CUDA(c, cudaMemcpyAsync(pot, d_pot, sizeof(double) * n_i, cudaMemcpyDeviceToHost, c->stream));
    NB_CUDA(c, cudaMemcpyAsync(nnb, c->st_nnb, sizeof(int32_t) * n_i, cudaMemcpyDeviceToHost, c->stream));
    NB_CUDA(c, cudaMemcpyAsync(overflow, c->st_ovf, sizeof(int32_t) * n_i, cudaMemcpyDeviceToHost, c->stream));
    NB_CUDA(c, cudaStreamSynchronize(c->stream));
    if (nblist) {
        // only the first min(nnb, cap) entries of a row are defined: copy the columns some row uses
        // (a pitched copy of [n_i][maxc] out of [n_i][cap]; 150 of 512 columns in the headline config)
        int32_t maxc = 0;
        for (int32_t k = 0; k < n_i; ++k) maxc = std::max(maxc, std::min(nnb[k], c->cap));
        if (maxc > 0) {
            const size_t pitch = sizeof(int32_t) * (size_t)c->cap;
            NB_CUDA(c, cudaMemcpy2DAsync(nblist, pitch, c->st_list, pitch, sizeof(int32_t) * (size_t)maxc, (size_t)n_i,
                                         cudaMemcpyDeviceToHost, c->stream));
            NB_CUDA(c, cudaStreamSynchronize(c->stream));
        }
    }
    return NB_OK;
}

}  // namespace

extern "C" {

int nb_open(int64_t N, int32_t nb_cap, nb_ctx **out) {
    if (!out) return NB_EINVAL;
    *out = nullptr;
    if (N <= 0 || nb_cap <= 0 || N > (int64_t)1 << 30) return NB_EINVAL;
    nb_ctx *c = new (std::nothrow) nb_ctx();
    if (!c) return NB_ENOMEM;
    int dev = 0;
    cudaDeviceProp prop;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, dev);
    if (e != cudaSuccess || prop.major != 10) {   // sm_100a only, no fallback of any kind
        delete c;
        return NB_ECUDA;
    }
    c->N = N; c->cap = nb_cap; c->device = dev;
    c->Npad = (N + TJ - 1) / TJ * TJ;
    c->Ns = c->Npad;
    c->sm_count = prop.multiProcessorCount;
    *out = c;     // from here on nb_close() releases whatever was allocated
    NB_CUDA(c, cudaMalloc(&c->soa, sizeof(double) * 14 * c->Ns));
    NB_CUDA(c, cudaMemsetAsync(c->soa, 0, sizeof(double) * 14 * c->Ns, nullptr));
    if (c->Npad > c->N) {     // padding bodies: massless ghosts, written once
        ghost_pad_kernel<<<(unsigned)((c->Npad - c->N + 255) / 256), 256>>>(c->N, c->Npad, c->Ns, c->soa);
        NB_CUDA(c, cudaGetLastError());
    }
    NB_CUDA(c, cudaMalloc(&c->rec, sizeof(float) * RECF * c->Npad));
    NB_CUDA(c, cudaMalloc(&c->cnt, sizeof(int32_t) * c->N));
    NB_CUDA(c, cudaMemset(c->cnt, 0, sizeof(int32_t) * c->N));
    c->cnt_n = c->N;
    {   // ascending list rows: one warp per row, P ints of shared memory each (finalize_kernel)
        int P = 32;
        while (P < nb_cap) P <<= 1;
        c->sort_P = P;
        // The attribute is per function and per device, NOT per context: every nb_open sets the same fixed
        // maximum, so a later context with a smaller cap cannot lower the limit under an older one.
        c->sort_smem_max = 200 * 1024;
        NB_CUDA(c, cudaFuncSetAttribute(finalize_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->sort_smem_max));
        NB_CUDA(c, cudaFuncSetAttribute(finalize_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->sort_smem_max));
    }
    NB_CUDA(c, (setup_variant<8, 1, 2>(c->var[0], VAR_OVH[0])));
    NB_CUDA(c, (setup_variant<4, 2, 2>(c->var[1], VAR_OVH[1])));
    NB_CUDA(c, (setup_variant<2, 4, 2>(c->var[2], VAR_OVH[2])));
    NB_CUDA(c, (setup_variant<1, 8, 2>(c->var[3], VAR_OVH[3])));
    NB_CUDA(c, (setup_variant<1, 8, 2, true>(c->var[4], VAR_OVH[4])));
    NB_CUDA(c, (setup_variant<2, 4, 2, false, SRC_STATE>(c->fvar[2], VAR_OVH[2])));
    NB_CUDA(c, (setup_variant<1, 8, 2, false, SRC_STATE>(c->fvar[3], VAR_OVH[3])));
    NB_CUDA(c, (setup_variant<1, 8, 2, true, SRC_STATE>(c->fvar[4], VAR_OVH[4])));
    NB_CUDA(c, cudaStreamSynchronize(nullptr));     // the ghost padding is in place before any stream uses the state
    return NB_OK;
}

int nb_close(nb_ctx *c) {
    if (!c) return NB_EINVAL;
    cudaStreamSynchronize(c->stream);
    cudaFree(c->soa); cudaFree(c->aos); cudaFree(c->rec); cudaFree(c->cnt); cudaFree(c->stats);
    cudaFree(c->sort_keys); cudaFree(c->sort_box);
    cudaFree(c->blk_key); cudaFree(c->blk_idx); cudaFree(c->blk_out); cudaFree(c->blk_nnb); cudaFree(c->blk_ovf);
    cudaFree(c->blk_list);
    cudaFree(c->ac.aI); cudaFree(c->ac.jI); cudaFree(c->ac.aR); cudaFree(c->ac.jR); cudaFree(c->ac.tR); cudaFree(c->ac.dtR);
    cudaFree(c->ac.nnb); cudaFree(c->ac.list); cudaFree(c->ac_h2); cudaFree(c->ac_aIo); cudaFree(c->ac_jIo);
    cudaFree(c->ac_reg_idx); cudaFree(c->ac_novf); cudaFree(c->ac_in); cudaFreeHost(c->h_ac_novf);
    cudaFree(c->blk_stall); cudaFree(c->blk_pub); cudaFree(c->sel_cmin); cudaFree(c->sel_dirty); cudaFree(c->p64); cudaFreeHost(c->h_blk_ring);
    cudaFree(c->partial); cudaFree(c->stage_j);
    cudaFree(c->st_idx); cudaFree(c->st_nnb); cudaFree(c->st_ovf); cudaFree(c->st_list);
    cudaFree(c->st_h2); cudaFree(c->st_out);
    cudaFree(c->d_ist); cudaFree(c->irec); cudaFreeHost(c->h_ist);
    cudaFree(c->dtj); cudaFree(c->sel_key); cudaFree(c->sel_counts); cudaFree(c->sel_result);
    cudaFreeHost(c->h_sel_result);
    if (c->ev_enter) cudaEventDestroy(c->ev_enter);
    if (c->ev_i) cudaEventDestroy(c->ev_i);
    for (int q = 0; q < nb_ctx::MAXCHUNK; ++q) {
        if (c->ev_chunk[q]) cudaEventDestroy(c->ev_chunk[q]);
        if (c->ev_copied[q]) cudaEventDestroy(c->ev_copied[q]);
    }
    for (int q = 0; q < nb_ctx::MAXCHUNK; ++q) {
        if (c->force_stream[q]) cudaStreamDestroy(c->force_stream[q]);
        if (c->ev_force[q]) cudaEventDestroy(c->ev_force[q]);
    }
    if (c->ev_iready) cudaEventDestroy(c->ev_iready);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    if (c->prep_stream) cudaStreamDestroy(c->prep_stream);
    for (int q = 0; q < nb_ctx::PROF_RING; ++q) {
        if (c->ev0[q]) cudaEventDestroy(c->ev0[q]);
        if (c->ev1[q]) cudaEventDestroy(c->ev1[q]);
    }
    delete c;
    return NB_OK;
}

int nb_set_stream(nb_ctx *c, void *cuda_stream) {
    int rc = check_live(c);
    if (rc != NB_OK) return rc;
    c->stream = static_cast<cudaStream_t>(cuda_stream);
    return NB_OK;
}

int nb_synchronize(nb_ctx *c) {
    int rc = check_live(c);
    if (rc != NB_OK) return rc;
    NB_CUDA(c, cudaStreamSynchronize(c->stream));
    return NB_OK;
}

int nb_set_j(nb_ctx *c, const double *m, const double *x0, const double *v0, const double *a0, const double *j0,
             const double *t0) {
    int rc = check_live(c);
    if (rc != NB_OK) return rc;
    if (!m || !x0 || !v0 || !a0 || !j0 || !t0) return NB_EINVAL;
    relayout_kernel<<<(unsigned)((c->N + 255) / 256), 256, 0, c->stream>>>(0, c->N, c->Ns, m, x0, v0, a0, j0, t0, c->soa,
                                                                           c->aos);
    NB_CUDA(c, cudaGetLastError());
    c->launches += 1;
    c->have_j = true;
    c->sel_all_dirty = true;    // t0 changed: the per-chunk minima of t0 + dt are stale
    c->have_pred = false; c->pred_pending = false;
    c->have_ac = false;         // the AC force polynomials belong to the state that was just replaced
    return NB_OK;
}

int nb_set_j_host(nb_ctx *c, const double *m, const double *x0, const double *v0, const double *a0,
                  const double *j0, const double *t0) {
    int rc = check_live(c);
    if (rc != NB_OK) return rc;
    if (!m || !x0 || !v0 || !a0 || !j0 || !t0) return NB_EINVAL;
    const int64_t N = c->N;
    if (!c->stage_j) NB_CUDA(c, cudaMalloc(&c->stage_j, sizeof(double) * 14 * N));
    double *d = c->stage_j;
    double *dm = d, *dx = d + N, *dv = d + 4 * N, *da = d + 7 * N, *dj = d + 10 * N, *dt = d + 13 * N;
    NB_CUDA(c, cudaMemcpyAsync(dm, m, sizeof(double) * N, cudaMemcpyHostToDevice, c->stream));
    NB_CUDA(c, cudaMemcpyAsync(dx, x0, sizeof(double) * 3 * N, cudaMemcpyHostToDevice, c->stream));
    NB_CUDA(c, cudaMemcpyAsync(dv, v0, sizeof(double) * 3 * N, cudaMemcpyHostToDevice, c->stream));
    NB_CUDA(c, cudaMemcpyAsync(da, a0, sizeof(double) * 3 * N, cudaMemcpyHostToDevice, c->stream));
    NB_CUDA(c, cudaMemcpyAsync(dj, j0, sizeof(double) * 3 * N, cudaMemcpyHostToDevice, c->stream));
    NB_CUDA(c, cudaMemcpyAsync(dt, t0, sizeof(double) * N, cudaMemcpyHostToDevice, c->stream));
    return nb_set_j(c, dm, dx, dv, da, dj, dt);
}

int nb_update_j(nb_ctx *c, int32_t n, const int32_t *idx, const double *m, const double *x0, const double *v0,
                const double *a0, const double *j0, const double *t0) {
    int rc = check_live(c);
    if (rc != NB_OK) return rc;
    if (n < 0 || n > c->N) return NB_EINVAL;
    if (!c->have_j) return NB_ESTATE;
    if (n == 0) return NB_OK;
    if (!idx || !m || !x0 || !v0 || !a0 || !j0 || !t0) return NB_EINVAL;
    update_j_kernel<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(n, c->Ns, idx, m, x0, v0, a0, j0, t0, c->soa,
                                                                         c->aos);
    NB_CUDA(c, cudaGetLastError());
    c->launches += 1;
    c->have_pred = false; c->pred_pending = false;   // the predicted records are stale until the next nb_predict_all
    c->sel_all_dirty = true;
    c->have_ac = false;
    return NB_OK;
}

int nb_irregular(nb_ctx *c, double t, int32_t n_i, const int32_t *idx_i, const int32_t *nnb, const int32_t *nblist,
                 double *acc, double *jerk, double *pot) {
    int rc = check_live(c);
    if (rc != NB_OK) return rc;
    if (n_i < 0 || n_i > c->N) return NB_EINVAL;
    if (!c->have_j) return NB_ESTATE;
    if (n_i == 0) return NB_OK;
    if (!idx_i || !nnb || !nblist || !acc || !jerk) return NB_EINVAL;
    rc = ensure_aos(c);
    if (rc != NB_OK) return rc;
    return launch_irregular<false>(c, false, n_i, t, nullptr, 0, 0, idx_i, nnb, nblist, acc, jerk, pot);
}

int nb_predict_all(nb_ctx *c, double t) {
    int rc = check_live(c);
    if (rc != NB_OK) return rc;
    if (!c->have_j) return NB_ESTATE;
    // The launch is deferred: a small block that follows predicts inside its force kernel (fused path) and
    // never needs the records; any other consumer writes them first (materialize_pred).  The result of
    // every later call is the same either way.
    c->have_pred = true;
    c->pred_pending = true;
    c->pred_t = t;
    return c->fuse ? NB_OK : materialize_pred(c);
}

int nb_get_predicted(nb_ctx *c, double *xp, double *vp) {
    int rc = check_live(c);
    if (rc != NB_OK) return rc;
    if (!xp || !vp) return NB_EINVAL;
    if (!c->have_pred) return NB_ESTATE;
    rc = materialize_pred(c);
    if (rc != NB_OK) return rc;
    unpack_predicted_kernel<<<(unsigned)((c->N + 255) / 256), 256, 0, c->stream>>>(c->N, c->rec, xp, vp);
    NB_CUDA(c, cudaGetLastError());
    c->launches += 1;
    return NB_OK;
}

int nb_regular(nb_ctx *c, int32_t n_i, const int32_t *idx_i, const double *h2_i, double *acc, double *jerk,
               double *pot, int32_t *nnb, int32_t *nblist, int32_t *overflow) {
    int rc = check_live(c);
    if (rc != NB_OK) return rc;
    if (n_i < 0 || n_i > c->N) return NB_EINVAL;
    if (!c->have_pred) return NB_ESTATE;
    if (n_i == 0) return NB_OK;
    if (!idx_i || !h2_i || !acc || !jerk || !pot || !nnb || !nblist || !overflow) return NB_EINVAL;
    return regular_device(c, n_i, idx_i, h2_i, acc, jerk, pot, nnb, nblist, overflow);
}

int nb_regular_all(nb_ctx *c, const double *h2, double *acc, double *jerk, double *pot, int32_t *nnb,
                   int32_t *nblist, int32_t *overflow) {
    int rc = check_live(c);
    if (rc != NB_OK) return rc;
    if (!c->have_pred) return NB_ESTATE;
    if (!h2 || !acc || !jerk || !pot || !nnb || !overflow) return NB_EINVAL;
    return regular_device(c, (int32_t)c->N, nullptr, h2, acc, jerk, pot, nnb, nblist, overflow);
}

int nb_regular_host(nb_ctx *c, int32_t n_i, const int32_t *idx_i, const double *h2_i, double *acc, double *jerk,
                    double *pot, int32_t *nnb, int32_t *nblist, int32_t *overflow) {
    int rc = check_live(c);
    if (rc != NB_OK) return rc;
    if (n_i < 0 || n_i > c->N) return NB_EINVAL;
    if (!c->have_pred) return NB_ESTATE;
    if (n_i == 0) return NB_OK;
    if (!idx_i || !h2_i || !acc || !jerk || !pot || !nnb || !overflow) return NB_EINVAL;
    rc = ensure_host_staging(c, n_i, true);
    if (rc != NB_OK) return rc;
    double *d_acc = c->st_out, *d_jerk = c->st_out + 3 * (int64_t)n_i, *d_pot = c->st_out + 6 * (int64_t)n_i;
    NB_CUDA(c, cudaMemcpyAsync(c->st_idx, idx_i, sizeof(int32_t) * n_i, cudaMemcpyHostToDevice, c->stream));
    NB_CUDA(c, cudaMemcpyAsync(c->st_h2, h2_i, sizeof(double) * n_i, cudaMemcpyHostToDevice, c->stream));
    rc = regular_device(c, n_i, c->st_idx, c->st_h2, d_acc, d_jerk, d_pot, c->st_nnb, c->st_list, c->st_ovf);
    if (rc != NB_OK) return rc;
    return copy_back(c, n_i, acc, jerk, pot, nnb, nblist, overflow);
}

int nb_step_host(nb_ctx *c, const double *m, const double *x0, const double *v0, const double *a0, const double *j0,
                 const double *t0, double t, int32_t n_i, const int32_t *idx_i, const double *h2_i, double *acc,
                 double *jerk, double *pot, int32_t *nnb, int32_t *nblist, int32_t *overflow) {
    int rc = check_live(c);
    if (rc != NB_OK) return rc;
    if (!m || !x0 || !v0 || !a0 || !j0 || !t0) return NB_EINVAL;
    if (n_i < 0 || n_i > c->N) return NB_EINVAL;
    if (c->j_offset != 0) return NB_ESTATE;      // a shard context: blocks go through nb_regular_shard
    if (n_i == 0) {
        rc = nb_set_j_host(c, m, x0, v0, a0, j0, t0);
        if (rc == NB_OK) rc = nb_predict_all(c, t);
        if (rc == NB_OK) rc = nb_synchronize(c);
        return rc;
    }
    if (!idx_i || !h2_i || !acc || !jerk || !pot || !nnb || !overflow) return NB_EINVAL;
    for (int32_t k = 0; k < n_i; ++k)
        if (idx_i[k] < 0 || idx_i[k] >= c->N) return NB_EINVAL;      // the host has them in hand: checked here
    const int64_t N = c->N;
    if (!c->copy_stream) {
        NB_CUDA(c, cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
        NB_CUDA(c, cudaStreamCreateWithFlags(&c->prep_stream, cudaStreamNonBlocking));
        NB_CUDA(c, cudaEventCreateWithFlags(&c->ev_enter, cudaEventDisableTiming));
        NB_CUDA(c, cudaEventCreateWithFlags(&c->ev_i, cudaEventDisableTiming));
        for (int q = 0; q < nb_ctx::MAXCHUNK; ++q) {
            NB_CUDA(c, cudaEventCreateWithFlags(&c->ev_chunk[q], cudaEventDisableTiming));
            NB_CUDA(c, cudaEventCreateWithFlags(&c->ev_copied[q], cudaEventDisableTiming));
        }
    }
    if (!c->stage_j) NB_CUDA(c, cudaMalloc(&c->stage_j, sizeof(double) * 14 * N));
    const int vi = pick_variant(c, n_i);
    const Variant &v = c->var[vi];
    const int64_t n_ib = (n_i + v.iblock - 1) / v.iblock;
    const int64_t n_i_pad = n_ib * v.iblock;
    rc = ensure_host_staging(c, n_i, true);
    if (rc != NB_OK) return rc;
    if (n_i_pad > c->ist_n) {
        NB_CUDA(c, cudaStreamSynchronize(c->stream));
        cudaFree(c->d_ist); cudaFree(c->irec); cudaFreeHost(c->h_ist);
        c->d_ist = nullptr; c->irec = nullptr; c->h_ist = nullptr; c->ist_n = 0;
        const int64_t n = std::max<int64_t>(n_i_pad, 1024) * 5 / 4;
        NB_CUDA(c, cudaMallocHost(&c->h_ist, sizeof(double) * 14 * n));
        NB_CUDA(c, cudaMalloc(&c->d_ist, sizeof(double) * 14 * n));
        NB_CUDA(c, cudaMalloc(&c->irec, sizeof(float) * RECF * n));
        c->ist_n = n;
    }
    // the active particles' own state must not wait for the chunk that holds it.  Pinned (mapped) host
    // arrays are gathered by the kernel itself through the bus; pageable ones by the host into a pinned
    // staging buffer (marshalling only: 14 doubles per active particle).
    IStateSrc isrc = {};
    bool zero_copy = true;
    {
        const void *hp[7] = {m, x0, v0, a0, j0, t0, idx_i};
        const void *dp[7];
        for (int q = 0; q < 7 && zero_copy; ++q) {
            cudaPointerAttributes at;
            if (cudaPointerGetAttributes(&at, hp[q]) != cudaSuccess) { cudaGetLastError(); zero_copy = false; break; }
            if (at.type != cudaMemoryTypeHost || !at.devicePointer) zero_copy = false;
            dp[q] = at.devicePointer;
        }
        if (zero_copy) {
            isrc.m = (const double *)dp[0]; isrc.x0 = (const double *)dp[1]; isrc.v0 = (const double *)dp[2];
            isrc.a0 = (const double *)dp[3]; isrc.j0 = (const double *)dp[4]; isrc.t0 = (const double *)dp[5];
            isrc.idx_i = (const int32_t *)dp[6];
        }
    }
    if (!zero_copy) {
        double *h = c->h_ist;
        const size_t n = (size_t)n_i;
        for (size_t k = 0; k < n; ++k) {
            const int64_t i = idx_i[k];
            h[k] = m[i];
            h[13 * n + k] = t0[i];
            for (int q = 0; q < 3; ++q) {
                h[(1 + q) * n + k] = x0[3 * i + q];
                h[(4 + q) * n + k] = v0[3 * i + q];
                h[(7 + q) * n + k] = a0[3 * i + q];
                h[(10 + q) * n + k] = j0[3 * i + q];
            }
        }
        isrc.ist = c->d_ist;
    }
    // chunk plan: the j-range arrives as 1/16, 1/16, 1/8, 1/4, 1/2 of the tiles (first copy short,
    // every later copy hidden behind the force launches of the chunks before it)
    const int64_t ntiles = c->Npad / TJ;
    int64_t ctile[nb_ctx::MAXCHUNK + 1];
    const int nchunk = plan_chunks_pure(ntiles, c->step_chunks, ctile);
    int S_c[nb_ctx::MAXCHUNK], S_total = 0;
    for (int q = 0; q < nchunk; ++q) {
        S_c[q] = pick_split(c, v, n_ib, ctile[q + 1] - ctile[q]);
        S_total += S_c[q];
    }
    rc = ensure_partial(c, (size_t)S_total * 7 * n_i_pad * sizeof(double));
    if (rc != NB_OK) return rc;

    cudaStream_t cs = c->copy_stream, ps = c->prep_stream;
    NB_CUDA(c, cudaEventRecord(c->ev_enter, c->stream));          // staging buffers are free once earlier work ran
    NB_CUDA(c, cudaStreamWaitEvent(cs, c->ev_enter, 0));
    NB_CUDA(c, cudaStreamWaitEvent(ps, c->ev_enter, 0));
    NB_CUDA(c, cudaMemcpyAsync(c->st_idx, idx_i, sizeof(int32_t) * n_i, cudaMemcpyHostToDevice, cs));
    NB_CUDA(c, cudaMemcpyAsync(c->st_h2, h2_i, sizeof(double) * n_i, cudaMemcpyHostToDevice, cs));
    if (!zero_copy)
        NB_CUDA(c, cudaMemcpyAsync(c->d_ist, c->h_ist, sizeof(double) * 14 * n_i, cudaMemcpyHostToDevice, cs));
    NB_CUDA(c, cudaEventRecord(c->ev_i, cs));
    double *d = c->stage_j;
    double *dm = d, *dx = d + N, *dv = d + 4 * N, *da = d + 7 * N, *dj = d + 10 * N, *dt0 = d + 13 * N;
    for (int q = 0; q < nchunk; ++q) {
        const int64_t jb = ctile[q] * TJ, je_pad = ctile[q + 1] * TJ, je = std::min<int64_t>(je_pad, N);
        const size_t n1 = sizeof(double) * (size_t)(je - jb), n3 = 3 * n1;
        if (je > jb) {
            NB_CUDA(c, cudaMemcpyAsync(dm + jb, m + jb, n1, cudaMemcpyHostToDevice, cs));
            NB_CUDA(c, cudaMemcpyAsync(dx + 3 * jb, x0 + 3 * jb, n3, cudaMemcpyHostToDevice, cs));
            NB_CUDA(c, cudaMemcpyAsync(dv + 3 * jb, v0 + 3 * jb, n3, cudaMemcpyHostToDevice, cs));
            NB_CUDA(c, cudaMemcpyAsync(da + 3 * jb, a0 + 3 * jb, n3, cudaMemcpyHostToDevice, cs));
            NB_CUDA(c, cudaMemcpyAsync(dj + 3 * jb, j0 + 3 * jb, n3, cudaMemcpyHostToDevice, cs));
            NB_CUDA(c, cudaMemcpyAsync(dt0 + jb, t0 + jb, n1, cudaMemcpyHostToDevice, cs));
            // the kernels of a landed chunk go to their own stream: they may wait for SM slots behind the
            // running force launch, and the next chunk's copies must not queue behind them
            NB_CUDA(c, cudaEventRecord(c->ev_copied[q], cs));
            NB_CUDA(c, cudaStreamWaitEvent(ps, c->ev_copied[q], 0));
            relayout_kernel<<<(unsigned)((je - jb + 255) / 256), 256, 0, ps>>>(jb, je, c->Ns, dm, dx, dv, da, dj, dt0,
                                                                               c->soa, c->aos);
        }
        predict_kernel<<<(unsigned)((je_pad - jb + 255) / 256), 256, 0, ps>>>(jb, je_pad, N, c->Ns, t, c->soa, c->rec);
        NB_CUDA(c, cudaGetLastError());
        NB_CUDA(c, cudaEventRecord(c->ev_chunk[q], ps));
        c->launches += 2;
    }
    c->have_j = true;
    c->sel_all_dirty = true;
    c->have_pred = true; c->pred_pending = false;     // every chunk is predicted as it lands
    c->pred_t = t;

    NB_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_i, 0));
    if (zero_copy)
        predict_i_kernel<true><<<(unsigned)((n_i + 255) / 256), 256, 0, c->stream>>>(n_i, (int32_t)n_i_pad, t, isrc, c->irec);
    else
        predict_i_kernel<false><<<(unsigned)((n_i + 255) / 256), 256, 0, c->stream>>>(n_i, (int32_t)n_i_pad, t, isrc, c->irec);
    NB_CUDA(c, cudaGetLastError());
    c->launches += 1;
    const unsigned long long *perm = nullptr;
    c->last_reordered = 0;
    if (want_reorder(c, n_i)) {        // from the active particles' own records: no chunk of the j-state is needed
        rc = reorder_block(c, n_i, c->st_idx, c->irec, n_i_pad);
        if (rc != NB_OK) return rc;
        perm = c->sort_keys; c->last_reordered = 1;
    }
    // The per-chunk force launches are independent (own partial rows; the row counters are integer atomics): each
    // goes to its own stream behind its chunk's predictor, so that the CTAs of a chunk fill the drain of the one
    // before it instead of queueing behind its last CTA.
    if (!c->force_stream[0]) {
        for (int q = 0; q < nb_ctx::MAXCHUNK; ++q) {
            NB_CUDA(c, cudaStreamCreateWithFlags(&c->force_stream[q], cudaStreamNonBlocking));
            NB_CUDA(c, cudaEventCreateWithFlags(&c->ev_force[q], cudaEventDisableTiming));
        }
        NB_CUDA(c, cudaEventCreateWithFlags(&c->ev_iready, cudaEventDisableTiming));
    }
    NB_CUDA(c, cudaEventRecord(c->ev_iready, c->stream));       // i-records, Morton order, scratch: ready
    int64_t split0 = 0;
    for (int q = 0; q < nchunk; ++q) {
        cudaStream_t fs = c->force_stream[q];
        NB_CUDA(c, cudaStreamWaitEvent(fs, c->ev_iready, 0));
        NB_CUDA(c, cudaStreamWaitEvent(fs, c->ev_chunk[q], 0));
        rc = launch_force_range(c, vi, false, n_i, c->st_idx, c->st_h2, c->irec, perm, 0, c->st_list, ctile[q], ctile[q + 1], S_c[q],
                                split0, fs, false);
        if (rc != NB_OK) return rc;
        NB_CUDA(c, cudaEventRecord(c->ev_force[q], fs));
        NB_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_force[q], 0));
        split0 += S_c[q];
    }
    double *d_acc = c->st_out, *d_jerk = c->st_out + 3 * (int64_t)n_i, *d_pot = c->st_out + 6 * (int64_t)n_i;
    rc = launch_finalize(c, n_i, n_i_pad, S_total, perm, d_acc, d_jerk, d_pot, c->st_nnb, c->st_list, c->st_ovf);
    if (rc != NB_OK) return rc;
    rc = copy_back(c, n_i, acc, jerk, pot, nnb, nblist, overflow);
    return rc;
}

int nb_set_steps(nb_ctx *c, const double *dt) {
    int rc = check_live(c);
    if (rc != NB_OK) return rc;
    if (!dt) return NB_EINVAL;
    if (!c->have_j) return NB_ESTATE;
    if (!c->dtj) NB_CUDA(c, cudaMalloc(&c->dtj, sizeof(double) * c->N));
    NB_CUDA(c, cudaMemcpyAsync(c->dtj, dt, sizeof(double) * c->N, cudaMemcpyDeviceToDevice, c->stream));
    c->have_steps = true;
    c->sel_all_dirty = true;
    c->have_ac = false;         // dtj is the irregular step of the two-level scheme: replaced here
    return NB_OK;
}

int nb_init_steps(nb_ctx *c, double eta_s, double dt_max) {
    int rc = check_live(c);
    if (rc != NB_OK) return rc;
    if (!(eta_s > 0.0) || !(dt_max > 0.0)) return NB_EINVAL;
    if (!c->have_j) return NB_ESTATE;
    if (!c->dtj) NB_CUDA(c, cudaMalloc(&c->dtj, sizeof(double) * c->N));
    init_steps_kernel<<<(unsigned)((c->N + 255) / 256), 256, 0, c->stream>>>(c->N, c->Ns, eta_s, dt_max, c->soa, c->dtj);
    NB_CUDA(c, cudaGetLastError());
    c->launches += 1;
    c->have_steps = true;
    c->sel_all_dirty = true;
    c->have_ac = false;
    return NB_OK;
}

int nb_next_block(nb_ctx *c, double *t_next, int32_t *n_act, int32_t *idx_act) {
    int rc = check_live(c);
    if (rc != NB_OK) return rc;
    if (!t_next || !n_act || !idx_act) return NB_EINVAL;
    if (!c->have_j || !c->have_steps) return NB_ESTATE;
    const int64_t N = c->N;
    const unsigned nchunk = (unsigned)((N + SEL_CHUNK - 1) / SEL_CHUNK);
    if (!c->sel_key) {
        NB_CUDA(c, cudaMalloc(&c->sel_key, sizeof(unsigned long long)));
        NB_CUDA(c, cudaMalloc(&c->sel_counts, sizeof(int32_t) * nchunk));
        NB_CUDA(c, cudaMalloc(&c->sel_result, sizeof(double) * 4));
        NB_CUDA(c, cudaMallocHost(&c->h_sel_result, sizeof(double) * 4));
    }
    const double *t0 = c->soa + 13 * c->Ns;
    NB_CUDA(c, cudaMemsetAsync(c->sel_key, 0xff, sizeof(unsigned long long), c->stream));
    const unsigned g = (unsigned)std::min<int64_t>((N + 255) / 256, (int64_t)c->sm_count * 8);
    next_time_kernel<<<g, 256, 0, c->stream>>>(N, t0, c->dtj, c->sel_key);
    select_active_kernel<0><<<nchunk, 256, 0, c->stream>>>(N, t0, c->dtj, c->sel_key, c->sel_counts, idx_act, c->sel_result);
    select_active_kernel<1><<<nchunk, 256, 0, c->stream>>>(N, t0, c->dtj, c->sel_key, c->sel_counts, idx_act, c->sel_result);
    NB_CUDA(c, cudaGetLastError());
    c->launches += 3;
    NB_CUDA(c, cudaMemcpyAsync(c->h_sel_result, c->sel_result, sizeof(double) * 2, cudaMemcpyDeviceToHost, c->stream));
    NB_CUDA(c, cudaStreamSynchronize(c->stream));
    *t_next = c->h_sel_result[0];
    *n_act = (int32_t)c->h_sel_result[1];
    return NB_OK;
}

int nb_correct(nb_ctx *c, double t, int32_t n, const int32_t *idx, const double *acc1, const double *jerk1,
               double eta, double dt_max) {
    int rc = check_live(c);
    if (rc != NB_OK) return rc;
    if (n < 0 || n > c->N || !(eta > 0.0) || !(dt_max > 0.0)) return NB_EINVAL;
    if (!c->have_j || !c->have_steps) return NB_ESTATE;
    if (n == 0) return NB_OK;
    if (!idx || !acc1 || !jerk1) return NB_EINVAL;
    rc = ensure_aos(c);
    if (rc != NB_OK) return rc;
    correct_kernel<<<(unsigned)((n + 127) / 128), 128, 0, c->stream>>>(n, c->Ns, t, eta, dt_max, nullptr, idx, acc1,
                                                                       jerk1, c->soa, c->aos, c->dtj, c->sel_dirty);
    NB_CUDA(c, cudaGetLastError());
    c->launches += 1;
    c->have_pred = false; c->pred_pending = false;
    c->have_ac = false;         // the single-level corrector knows nothing of the AC force polynomials
    return NB_OK;
}

}  // extern "C"

namespace {

// ---------------------------------------------------------------------------------------------------------
// The block loop (nb_block_step / nb_run_blocks, nb_ac_step / nb_ac_run): ONE engine.  A BATCH of blocks is
// enqueued without the host in between: per block the cooperative selection kernel, then the chain that can
// integrate a small block with {t, n} taken from device memory (speculative: a no-op unless the selection
// marked the block BLK_SPECULATIVE).  The first block of a batch that needs the host (too large, a regular
// step due, past t_stop) sets the device stall flag; the rest of the batch does nothing and that block's lists
// stay in place.  The host reads the batch's descriptors once, finishes the stalled block by the ordinary
// launches, and enqueues the next batch.
constexpr int BLK_BATCH_MAX = 16;
constexpr int32_t AC_SPEC_CAP = 1024;

int blk_setup(nb_ctx *c) {
    if (c->blk_key) return NB_OK;
    const int64_t N = c->N;
    const int nchunk = (int)((N + SEL_CHUNK - 1) / SEL_CHUNK);
    NB_CUDA(c, cudaMalloc(&c->blk_key, 2 * sizeof(unsigned long long)));
    NB_CUDA(c, cudaMemsetAsync(c->blk_key, 0xff, 2 * sizeof(unsigned long long), c->stream));
    NB_CUDA(c, cudaMalloc(&c->blk_idx, sizeof(int32_t) * std::max<int64_t>(N, 1024)));   // (speculative launches read up to their capacity)
    NB_CUDA(c, cudaMalloc(&c->ac_reg_idx, sizeof(int32_t) * N));
    NB_CUDA(c, cudaMalloc(&c->blk_pub, sizeof(unsigned long long) * nchunk));
    NB_CUDA(c, cudaMemsetAsync(c->blk_pub, 0, sizeof(unsigned long long) * nchunk, c->stream));
    if (!c->sel_result) NB_CUDA(c, cudaMalloc(&c->sel_result, sizeof(double) * 4));
    if (!c->h_sel_result) NB_CUDA(c, cudaMallocHost(&c->h_sel_result, sizeof(double) * 4));
    // the descriptors of a batch live in MAPPED pinned host memory: the selection kernel stores them there itself
    // (status word last, after a system-wide fence), the host polls -- no copy operation or event in the stream
    NB_CUDA(c, cudaHostAlloc(&c->h_blk_ring, sizeof(double) * 4 * BLK_BATCH_MAX, cudaHostAllocMapped));
    NB_CUDA(c, cudaHostGetDevicePointer(reinterpret_cast<void **>(&c->blk_ring), c->h_blk_ring, 0));
    NB_CUDA(c, cudaMalloc(&c->blk_stall, sizeof(int32_t)));
    NB_CUDA(c, cudaMalloc(&c->sel_cmin, sizeof(unsigned long long) * nchunk));
    NB_CUDA(c, cudaMalloc(&c->sel_dirty, sizeof(int32_t) * nchunk));
    c->sel_all_dirty = true;
    // the scatter kernel's look-back needs every CTA it may wait for to be resident: the grid never exceeds what the
    // device holds at once (each CTA then walks several chunks, ascending)
    int occ_two = 0, occ_one = 0;
    NB_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_two, select_scatter_kernel<true>, 256, 0));
    NB_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_one, select_scatter_kernel<false>, 256, 0));
    c->sel_grid_max = (int64_t)std::max(1, std::min(occ_two, occ_one)) * c->sm_count;
    return NB_OK;
}

// buffers of a block of n bodies (the speculative chains use them: they exist before anything is enqueued)
int blk_buffers(nb_ctx *c, int64_t n, bool lists, bool ac) {
    const int64_t N = c->N;
    const int64_t m = std::min<int64_t>(std::max<int64_t>(N, 1024), std::max<int64_t>(n, 1024) * 5 / 4);
    if (n > c->blk_n) {
        NB_CUDA(c, cudaStreamSynchronize(c->stream));
        cudaFree(c->blk_out); cudaFree(c->blk_nnb); cudaFree(c->blk_ovf);
        c->blk_out = nullptr; c->blk_nnb = c->blk_ovf = nullptr; c->blk_n = 0;
        NB_CUDA(c, cudaMalloc(&c->blk_out, sizeof(double) * 7 * m));
        NB_CUDA(c, cudaMalloc(&c->blk_nnb, sizeof(int32_t) * m));
        NB_CUDA(c, cudaMalloc(&c->blk_ovf, sizeof(int32_t) * m));
        c->blk_n = m;
    }
    if (lists && n * c->cap > c->blk_list_n) {
        NB_CUDA(c, cudaStreamSynchronize(c->stream));
        cudaFree(c->blk_list); c->blk_list = nullptr; c->blk_list_n = 0;
        NB_CUDA(c, cudaMalloc(&c->blk_list, sizeof(int32_t) * m * c->cap));
        c->blk_list_n = m * c->cap;
    }
    if (ac && n > c->ac_in_n) {
        NB_CUDA(c, cudaStreamSynchronize(c->stream));
        cudaFree(c->ac_in); c->ac_in = nullptr; c->ac_in_n = 0;
        NB_CUDA(c, cudaMalloc(&c->ac_in, sizeof(double) * 6 * m));
        c->ac_in_n = m;
    }
    return NB_OK;
}

// selection of the next block into blk_idx (and ac_reg_idx), descriptor into sel_result and ring slot `slot`
int blk_enqueue_select(nb_ctx *c, bool two, double t_stop, int32_t spec_cap, int slot) {
    const int64_t N = c->N;
    const double *t0 = c->soa + 13 * c->Ns;
    unsigned long long *key = c->blk_key + c->blk_parity, *key_next = c->blk_key + (1 - c->blk_parity);
    double *ring = c->blk_ring + 4 * slot;
    const unsigned nchunk = (unsigned)((N + SEL_CHUNK - 1) / SEL_CHUNK);
    const unsigned gmin = (unsigned)std::min<int64_t>((N + 255) / 256, (int64_t)c->sm_count * 8);
    c->blk_epoch += 1;
    const unsigned long long *cmin = c->sel_chunks ? c->sel_cmin : nullptr;
    const unsigned gscat = (unsigned)std::min<int64_t>(nchunk, c->sel_grid_cap > 0 ? std::min(c->sel_grid_cap, c->sel_grid_max)
                                                                                     : c->sel_grid_max);
    if (c->sel_chunks) {
        if (c->sel_all_dirty) {       // any non-zero word means "rescan"
            NB_CUDA(c, cudaMemsetAsync(c->sel_dirty, 1, sizeof(int32_t) * nchunk, c->stream));
            c->sel_all_dirty = false;
        }
        NB_CUDA(c, launch_chain(select_min_chunks_kernel, dim3(nchunk), dim3(256), 0, c->stream, N, t0, c->dtj, c->sel_cmin,
                                c->sel_dirty, key, key_next, c->blk_stall, ring));
    } else {
        c->sel_all_dirty = true;      // the per-chunk minima are not maintained on this route
        NB_CUDA(c, launch_chain(select_min_kernel, dim3(gmin), dim3(256), 0, c->stream, N, t0, c->dtj, key, key_next, c->blk_stall, ring));
    }
    if (two)
        NB_CUDA(c, launch_chain(select_scatter_kernel<true>, dim3(gscat), dim3(256), 0, c->stream, N, t0, c->dtj, key, c->blk_pub,
                                c->blk_epoch, c->blk_idx, c->sel_result, c->ac.tR, c->ac.dtR, c->ac_reg_idx, t_stop, spec_cap,
                                c->blk_stall, ring, cmin, (int32_t)nchunk));
    else
        NB_CUDA(c, launch_chain(select_scatter_kernel<false>, dim3(gscat), dim3(256), 0, c->stream, N, t0, c->dtj, key, c->blk_pub,
                                c->blk_epoch, c->blk_idx, c->sel_result, nullptr, nullptr, c->ac_reg_idx, t_stop, spec_cap,
                                c->blk_stall, ring, cmin, (int32_t)nchunk));
    NB_CUDA(c, cudaGetLastError());
    c->blk_parity ^= 1;
    c->launches += 2;
    return NB_OK;
}

// Single-level chain of one block: a2-a7 [+ neighbour force added in place, P:49] + corrector.  spec_cap > 0:
// speculative (n, t from the device descriptor; buffers laid out for spec_cap bodies).
int sl_enqueue_chain(nb_ctx *c, const double *h2_all, double eta, double dt_max, int32_t n, double t, int32_t spec_cap) {
    const int64_t stride = spec_cap > 0 ? spec_cap : n;
    double *acc = c->blk_out, *jerk = c->blk_out + 3 * stride, *pot = c->blk_out + 6 * stride;
    c->spec_dev = spec_cap > 0 ? c->sel_result : nullptr;
    c->have_pred = true; c->pred_pending = true; c->pred_t = t;
    int rc = NB_OK;
    if (!c->fuse) rc = materialize_pred(c);
    c->h2_by_body = 1;
    if (rc == NB_OK)
        rc = regular_device(c, n, c->blk_idx, h2_all, acc, jerk, pot, c->blk_nnb, h2_all ? c->blk_list : nullptr, c->blk_ovf);
    c->h2_by_body = 0;
    if (rc == NB_OK && h2_all) {
        rc = launch_irregular<true>(c, true, n, t, c->spec_dev, 0, 0, c->blk_idx, c->blk_nnb, c->blk_list, acc, jerk, pot);
    }
    if (rc == NB_OK) {
        launch_chain(correct_kernel, dim3((unsigned)((n + 127) / 128)), dim3(128), 0, c->stream, n, c->Ns, t, eta, dt_max, c->spec_dev,
                     c->blk_idx, acc, jerk, c->soa, c->aos, c->dtj, c->sel_dirty);
        c->launches += 1;
        if (cudaGetLastError() != cudaSuccess) { c->cuda_err = cudaErrorUnknown; rc = NB_ECUDA; }
    }
    c->spec_dev = nullptr;
    c->have_pred = false; c->pred_pending = false;
    c->blk_stride = stride;
    return rc;
}

// Two-level chain of a block WITHOUT a regular step (speculative or not): neighbour force over the lists, corrector.
int ac_enqueue_irregular_chain(nb_ctx *c, double eta_I, double eta_R, double dt_max, int32_t n, double t, bool spec) {
    const double *dev = spec ? c->sel_result : nullptr;
    int rc = launch_irregular<false>(c, true, n, t, dev, 1, 1, c->blk_idx, c->ac.nnb, c->ac.list, c->ac_aIo, c->ac_jIo, nullptr);
    if (rc != NB_OK) return rc;
    NB_CUDA(c, launch_chain(ac_correct_kernel, dim3((unsigned)((n + 127) / 128)), dim3(128), 0, c->stream, n, c->Ns, t, eta_I, eta_R,
                            dt_max, dev, c->blk_idx, c->ac_aIo, c->ac_jIo, 0, c->ac_reg_idx, nullptr, nullptr, nullptr, nullptr,
                            c->blk_nnb, c->ac, c->soa, c->aos, c->dtj, c->sel_dirty));
    NB_CUDA(c, cudaGetLastError());
    c->launches += 1;
    return NB_OK;
}

// Two-level block with nr > 0 regular steps, by the ordinary launches (the lists are in blk_idx / ac_reg_idx).
// *n_overflow > 0 and NB_EOVERFLOW: a new list overflowed; nothing was corrected (reading R38).
int ac_finish_block(nb_ctx *c, double eta_I, double eta_R, double dt_max, double t, int32_t n, int32_t nr, int32_t *n_overflow) {
    *n_overflow = 0;
    int rc = blk_buffers(c, nr, true, true);
    if (rc != NB_OK) return rc;
    rc = launch_irregular<false>(c, false, n, t, nullptr, 1, 1, c->blk_idx, c->ac.nnb, c->ac.list, c->ac_aIo, c->ac_jIo, nullptr);
    if (rc != NB_OK) return rc;
    const bool p64_ready = c->irr_pred_min > 0 && n >= c->irr_pred_min;      // the block's records are in place (nr <= n)
    double *rg_acc = c->blk_out, *rg_jerk = c->blk_out + 3 * (int64_t)nr, *rg_pot = c->blk_out + 6 * (int64_t)nr;
    double *in_acc = c->ac_in, *in_jerk = c->ac_in + 3 * (int64_t)nr;
    c->have_pred = true; c->pred_pending = true; c->pred_t = t;
    if (!c->fuse) {
        rc = materialize_pred(c);
        if (rc != NB_OK) return rc;
    }
    c->h2_by_body = 1;
    rc = regular_device(c, nr, c->ac_reg_idx, c->ac_h2, rg_acc, rg_jerk, rg_pot, c->blk_nnb, c->blk_list, c->blk_ovf);
    c->h2_by_body = 0;
    c->have_pred = false; c->pred_pending = false;
    if (rc != NB_OK) return rc;
    rc = launch_irregular<false>(c, false, nr, t, nullptr, 0, 0, c->ac_reg_idx, c->blk_nnb, c->blk_list, in_acc, in_jerk, nullptr,
                                 p64_ready);
    if (rc != NB_OK) return rc;
    // a list that overflowed would break regular + irregular = total (R38): checked BEFORE anything is corrected
    NB_CUDA(c, cudaMemsetAsync(c->ac_novf, 0, sizeof(int32_t), c->stream));
    count_overflow_kernel<<<(unsigned)std::min<int64_t>((nr + 255) / 256, 1024), 256, 0, c->stream>>>(nr, c->blk_ovf, c->ac_novf);
    NB_CUDA(c, cudaMemcpyAsync(c->h_ac_novf, c->ac_novf, sizeof(int32_t), cudaMemcpyDeviceToHost, c->stream));
    NB_CUDA(c, cudaStreamSynchronize(c->stream));
    c->launches += 2;
    if (*c->h_ac_novf > 0) {
        *n_overflow = *c->h_ac_novf;
        return NB_EOVERFLOW;
    }
    ac_correct_kernel<<<(unsigned)((n + 127) / 128), 128, 0, c->stream>>>(n, c->Ns, t, eta_I, eta_R, dt_max, nullptr, c->blk_idx, c->ac_aIo,
                                                                          c->ac_jIo, nr, c->ac_reg_idx, rg_acc, rg_jerk, in_acc, in_jerk,
                                                                          c->blk_nnb, c->ac, c->soa, c->aos, c->dtj, c->sel_dirty);
    ac_store_rows_kernel<<<(unsigned)((nr + 7) / 8), 256, 0, c->stream>>>(nr, c->cap, c->ac_reg_idx, c->blk_nnb, c->blk_list, c->ac.list);
    NB_CUDA(c, cudaGetLastError());
    c->launches += 2;
    return NB_OK;
}

struct BlockRun {
    bool two;                         // two-level AC stepping
    const double *h2_all;             // single level: radii by body or NULL
    double eta, eta_R, dt_max, t_stop;
    int64_t max_blocks;
    // results
    double t_next = 0.0;
    int64_t blocks = 0, steps = 0, reg_steps = 0;
    int32_t last_n = 0, last_nr = 0, n_overflow = 0;
};

int run_blocks(nb_ctx *c, BlockRun &R) {
    int rc = blk_setup(c);
    if (rc != NB_OK) return rc;
    rc = blk_buffers(c, R.two ? 1 : 128, R.h2_all != nullptr, R.two);
    if (rc != NB_OK) return rc;
    rc = ensure_aos(c);
    if (rc != NB_OK) return rc;
    c->blk_last_n = 0;
    c->blk_last_two = R.two;
    while (R.blocks < R.max_blocks) {
        // speculative capacity of this batch: two-level: any block without a regular step up to AC_SPEC_CAP bodies;
        // single level: the size class of the last block (32 / 64 / 128: the variants with a fused predictor)
        int32_t spec_cap = 0;
        if (c->spec_enabled) {
            if (R.two) spec_cap = (int32_t)std::min<int64_t>(AC_SPEC_CAP, c->N);
            else if (c->fuse && c->blk_prev_n > 0 && c->blk_prev_n <= 128) {
                spec_cap = c->blk_prev_n <= 32 ? 32 : c->blk_prev_n <= 64 ? 64 : 128;
                // only if a block of that capacity takes the fused kernel (regular_device: one i-block of a variant that
                // has a fused form) -- NB_TUNE_FORCE_VARIANT can say otherwise, and then the block time must come
                // from the host: no speculation
                const int vi = pick_variant(c, spec_cap);
                if (vi < FUSED_FIRST || spec_cap > c->var[vi].iblock) spec_cap = 0;
            }
        }
        // batch size: 1 after a stall, doubled after every batch that ran without the host (a stalled batch wastes the
        // launches behind the stall)
        const int batch = (int)std::min<int64_t>(spec_cap > 0 ? c->blk_batch : 1, R.max_blocks - R.blocks);
        if (c->blk_stall_dirty) {
            NB_CUDA(c, cudaMemsetAsync(c->blk_stall, 0, sizeof(int32_t), c->stream));
            c->blk_stall_dirty = false;
        }
        volatile double *hring = c->h_blk_ring;
        for (int k = 0; k < batch; ++k) hring[4 * k + 3] = -1.0;          // "not written yet"
        for (int k = 0; k < batch; ++k) {
            rc = blk_enqueue_select(c, R.two, R.t_stop, spec_cap, k);
            if (rc != NB_OK) return rc;
            if (spec_cap > 0) {
                rc = R.two ? ac_enqueue_irregular_chain(c, R.eta, R.eta_R, R.dt_max, spec_cap, 0.0, true)
                           : sl_enqueue_chain(c, R.h2_all, R.eta, R.dt_max, spec_cap, 0.0, spec_cap);
                if (rc != NB_OK) return rc;
            }
        }
        // wait for the LAST selection's descriptor (not for the chain behind it); the stream is queried now and then
        // so that a failed launch cannot leave the host spinning
        for (uint64_t spin = 0; hring[4 * (batch - 1) + 3] < 0.0; ++spin) {
            if ((spin & 0xfff) == 0xfff) {
                const cudaError_t q = cudaStreamQuery(c->stream);
                if (q != cudaSuccess && q != cudaErrorNotReady) { c->cuda_err = q; return NB_ECUDA; }
                if (q == cudaSuccess && hring[4 * (batch - 1) + 3] < 0.0) { c->cuda_err = cudaErrorUnknown; return NB_ECUDA; }
            }
        }
        std::atomic_thread_fence(std::memory_order_acquire);
        bool stop = false;
        for (int k = 0; k < batch && !stop; ++k) {
            const double *d = c->h_blk_ring + 4 * k;
            const double t = d[0];
            const int32_t n = (int32_t)d[1], nr = (int32_t)d[2];
            const int status = (int)d[3];
            if (status == BLK_SKIPPED) break;                    // (cannot precede the block that stalled the batch)
            R.t_next = t;
            if (status == BLK_PAST_T_STOP || n <= 0) {                       // nothing is due before t_stop
                c->blk_stall_dirty = true; c->blk_batch = 1;
                return NB_OK;
            }
            if (status == BLK_SPECULATIVE) {
                c->spec_hits += 1;
            } else {                                             // BLK_NEEDS_HOST: the lists are in place, finish it here
                if (spec_cap > 0) c->spec_misses += 1;
                if (R.two) {
                    if (nr == 0) rc = ac_enqueue_irregular_chain(c, R.eta, R.eta_R, R.dt_max, n, t, false);
                    else {
                        rc = ac_finish_block(c, R.eta, R.eta_R, R.dt_max, t, n, nr, &R.n_overflow);
                        c->ac_fail_nr = rc == NB_EOVERFLOW ? nr : 0;       // rows and true counts stay in ac_reg_idx / blk_nnb
                    }
                } else {
                    rc = blk_buffers(c, n, R.h2_all != nullptr, false);
                    if (rc == NB_OK) rc = sl_enqueue_chain(c, R.h2_all, R.eta, R.dt_max, n, t, 0);
                }
                if (rc != NB_OK) { c->blk_stall_dirty = true; c->blk_batch = 1; return rc; }
                stop = true;                                     // the rest of the batch did nothing
            }
            R.blocks += 1; R.steps += n; R.reg_steps += nr;
            R.last_n = n; R.last_nr = nr;
            c->blk_prev_n = n;
            c->blk_last_n = n;
            c->blk_had_list = !R.two && R.h2_all != nullptr;
        }
        if (stop) { c->blk_stall_dirty = true; c->blk_batch = 1; }
        else if (spec_cap > 0) c->blk_batch = std::min(2 * c->blk_batch, BLK_BATCH_MAX);
    }
    return NB_OK;
}

}  // namespace

extern "C" {

int nb_block_step(nb_ctx *c, const double *h2_all, double eta, double dt_max, double t_stop, double *t_next,
                  int32_t *n_act) {
    int rc = check_live(c);
    if (rc != NB_OK) return rc;
    if (!t_next || !n_act || !(eta > 0.0) || !(dt_max > 0.0)) return NB_EINVAL;
    if (!c->have_j || !c->have_steps) return NB_ESTATE;
    BlockRun R = {false, h2_all, eta, 0.0, dt_max, t_stop, 1};
    c->have_ac = false;         // single-level steps leave the AC force polynomials behind
    rc = run_blocks(c, R);
    *t_next = R.t_next;
    *n_act = R.blocks ? R.last_n : 0;
    return rc;
}

int nb_run_blocks(nb_ctx *c, const double *h2_all, double eta, double dt_max, double t_stop, int64_t max_blocks,
                  double *t_next, int64_t *blocks, int64_t *particle_steps) {
    int rc = check_live(c);
    if (rc != NB_OK) return rc;
    if (!t_next || !blocks || !particle_steps || max_blocks < 0 || !(eta > 0.0) || !(dt_max > 0.0)) return NB_EINVAL;
    if (!c->have_j || !c->have_steps) return NB_ESTATE;
    BlockRun R = {false, h2_all, eta, 0.0, dt_max, t_stop, max_blocks};
    c->have_ac = false;
    rc = run_blocks(c, R);
    *t_next = R.t_next; *blocks = R.blocks; *particle_steps = R.steps;
    return rc;
}

int nb_ac_init(nb_ctx *c, double t_start, const double *h2_all, double eta_s, double dt_max, int32_t *n_overflow) {
    int rc = check_live(c);
    if (rc != NB_OK) return rc;
    if (!h2_all || !(eta_s > 0.0) || !(dt_max > 0.0)) return NB_EINVAL;
    if (!c->have_j) return NB_ESTATE;
    if (c->j_offset != 0) return NB_ESTATE;
    const int64_t N = c->N;
    if (!c->ac.aI) {
        const size_t v3 = sizeof(double) * 3 * N;
        NB_CUDA(c, cudaMalloc(&c->ac.aI, v3)); NB_CUDA(c, cudaMalloc(&c->ac.jI, v3));
        NB_CUDA(c, cudaMalloc(&c->ac.aR, v3)); NB_CUDA(c, cudaMalloc(&c->ac.jR, v3));
        NB_CUDA(c, cudaMalloc(&c->ac_aIo, v3)); NB_CUDA(c, cudaMalloc(&c->ac_jIo, v3));
        NB_CUDA(c, cudaMalloc(&c->ac.tR, sizeof(double) * N)); NB_CUDA(c, cudaMalloc(&c->ac.dtR, sizeof(double) * N));
        NB_CUDA(c, cudaMalloc(&c->ac_h2, sizeof(double) * N));
        NB_CUDA(c, cudaMalloc(&c->ac.nnb, sizeof(int32_t) * N));
        NB_CUDA(c, cudaMalloc(&c->ac.list, sizeof(int32_t) * N * c->cap));
        NB_CUDA(c, cudaMalloc(&c->ac_novf, sizeof(int32_t)));
        NB_CUDA(c, cudaMallocHost(&c->h_ac_novf, sizeof(int32_t)));
        if (!c->dtj) NB_CUDA(c, cudaMalloc(&c->dtj, sizeof(double) * N));
    }
    // every t0[j] must equal t_start (the start-up relabels x0, v0 as the state AT t_start): checked, because a call in
    // mid-run -- the tempting way out of an NB_EOVERFLOW -- would silently move every body that is not there
    NB_CUDA(c, cudaMemsetAsync(c->ac_novf, 0, sizeof(int32_t), c->stream));
    count_not_at_kernel<<<(unsigned)std::min<int64_t>((N + 255) / 256, (int64_t)c->sm_count * 8), 256, 0, c->stream>>>(
        N, c->soa + 13 * c->Ns, t_start, c->ac_novf);
    NB_CUDA(c, cudaGetLastError());
    c->launches += 1;
    NB_CUDA(c, cudaMemcpyAsync(c->h_ac_novf, c->ac_novf, sizeof(int32_t), cudaMemcpyDeviceToHost, c->stream));
    NB_CUDA(c, cudaStreamSynchronize(c->stream));
    if (*c->h_ac_novf != 0) return NB_ESTATE;
    rc = blk_setup(c);
    if (rc != NB_OK) return rc;
    c->ac_fail_nr = 0;
    NB_CUDA(c, cudaMemcpyAsync(c->ac_h2, h2_all, sizeof(double) * N, cudaMemcpyDeviceToDevice, c->stream));
    // forces at t_start: every t0[j] equals t_start, so the prediction is the state itself
    c->have_pred = true; c->pred_pending = true; c->pred_t = t_start;
    rc = ensure_aos(c);
    if (rc != NB_OK) return rc;
    int32_t *ovf_all = c->ac_reg_idx;               // scratch: free until the first step
    rc = regular_device(c, (int32_t)N, nullptr, c->ac_h2, c->ac.aR, c->ac.jR, c->ac_aIo /* pot: scratch */, c->ac.nnb,
                        c->ac.list, ovf_all);
    if (rc != NB_OK) return rc;
    rc = launch_irregular<false>(c, false, (int32_t)N, t_start, nullptr, 0, 0, nullptr, c->ac.nnb, c->ac.list, c->ac.aI, c->ac.jI,
                                 nullptr);
    if (rc != NB_OK) return rc;
    NB_CUDA(c, cudaMemsetAsync(c->ac_novf, 0, sizeof(int32_t), c->stream));
    ac_start_kernel<<<(unsigned)((N + 127) / 128), 128, 0, c->stream>>>(N, c->Ns, c->cap, t_start, eta_s, dt_max, c->ac, c->soa,
                                                                        c->aos, c->dtj, c->ac_novf);
    NB_CUDA(c, cudaGetLastError());
    c->launches += 2;
    NB_CUDA(c, cudaMemcpyAsync(c->h_ac_novf, c->ac_novf, sizeof(int32_t), cudaMemcpyDeviceToHost, c->stream));
    NB_CUDA(c, cudaStreamSynchronize(c->stream));
    c->have_pred = false; c->pred_pending = false;
    c->have_steps = true;
    c->sel_all_dirty = true;
    if (n_overflow) *n_overflow = *c->h_ac_novf;
    c->have_ac = *c->h_ac_novf == 0;
    return c->have_ac ? NB_OK : NB_EOVERFLOW;
}

int nb_ac_step(nb_ctx *c, double eta_I, double eta_R, double dt_max, double t_stop, double *t_next, int32_t *n_irr,
               int32_t *n_reg) {
    int rc = check_live(c);
    if (rc != NB_OK) return rc;
    if (!t_next || !n_irr || !n_reg || !(eta_I > 0.0) || !(eta_R > 0.0) || !(dt_max > 0.0)) return NB_EINVAL;
    if (!c->have_ac) return NB_ESTATE;
    BlockRun R = {true, nullptr, eta_I, eta_R, dt_max, t_stop, 1};
    rc = run_blocks(c, R);
    *t_next = R.t_next;
    *n_irr = R.blocks ? R.last_n : 0;
    *n_reg = rc == NB_EOVERFLOW ? R.n_overflow : (R.blocks ? R.last_nr : 0);
    return rc;
}

int nb_ac_run(nb_ctx *c, double eta_I, double eta_R, double dt_max, double t_stop, int64_t max_blocks, double *t_next,
              int64_t *blocks, int64_t *irregular_steps, int64_t *regular_steps) {
    int rc = check_live(c);
    if (rc != NB_OK) return rc;
    if (!t_next || !blocks || !irregular_steps || !regular_steps || max_blocks < 0) return NB_EINVAL;
    if (!(eta_I > 0.0) || !(eta_R > 0.0) || !(dt_max > 0.0)) return NB_EINVAL;
    if (!c->have_ac) return NB_ESTATE;
    BlockRun R = {true, nullptr, eta_I, eta_R, dt_max, t_stop, max_blocks};
    rc = run_blocks(c, R);
    *t_next = R.t_next; *blocks = R.blocks; *irregular_steps = R.steps; *regular_steps = R.reg_steps;
    return rc;
}

int nb_ac_get(nb_ctx *c, int32_t *idx_act, int32_t *idx_reg, double *aI, double *jI, double *aR, double *jR, double *tR,
              double *dtR, int32_t *nnb, int32_t *nblist) {
    int rc = check_live(c);
    if (rc != NB_OK) return rc;
    if (!c->ac.aI) return NB_ESTATE;
    const int64_t N = c->N;
    const cudaMemcpyKind dd = cudaMemcpyDeviceToDevice;
    if (idx_act) NB_CUDA(c, cudaMemcpyAsync(idx_act, c->blk_idx, sizeof(int32_t) * N, dd, c->stream));
    if (idx_reg) NB_CUDA(c, cudaMemcpyAsync(idx_reg, c->ac_reg_idx, sizeof(int32_t) * N, dd, c->stream));
    if (aI) NB_CUDA(c, cudaMemcpyAsync(aI, c->ac.aI, sizeof(double) * 3 * N, dd, c->stream));
    if (jI) NB_CUDA(c, cudaMemcpyAsync(jI, c->ac.jI, sizeof(double) * 3 * N, dd, c->stream));
    if (aR) NB_CUDA(c, cudaMemcpyAsync(aR, c->ac.aR, sizeof(double) * 3 * N, dd, c->stream));
    if (jR) NB_CUDA(c, cudaMemcpyAsync(jR, c->ac.jR, sizeof(double) * 3 * N, dd, c->stream));
    if (tR) NB_CUDA(c, cudaMemcpyAsync(tR, c->ac.tR, sizeof(double) * N, dd, c->stream));
    if (dtR) NB_CUDA(c, cudaMemcpyAsync(dtR, c->ac.dtR, sizeof(double) * N, dd, c->stream));
    if (nnb) NB_CUDA(c, cudaMemcpyAsync(nnb, c->ac.nnb, sizeof(int32_t) * N, dd, c->stream));
    if (nblist) NB_CUDA(c, cudaMemcpyAsync(nblist, c->ac.list, sizeof(int32_t) * N * c->cap, dd, c->stream));
    return NB_OK;
}

int nb_ac_set_radii(nb_ctx *c, int32_t n, const int32_t *idx, const double *h2) {
    int rc = check_live(c);
    if (rc != NB_OK) return rc;
    if (n < 0 || !h2 || (!idx && n != c->N)) return NB_EINVAL;
    if (!c->have_ac) return NB_ESTATE;
    if (n == 0) return NB_OK;
    if (!idx) {
        NB_CUDA(c, cudaMemcpyAsync(c->ac_h2, h2, sizeof(double) * c->N, cudaMemcpyDeviceToDevice, c->stream));
    } else {
        scatter_radii_kernel<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(n, c->N, idx, h2, c->ac_h2);
        NB_CUDA(c, cudaGetLastError());
        c->launches += 1;
    }
    return NB_OK;
}

int nb_ac_get_failed(nb_ctx *c, int32_t n_cap, int32_t *n_rows, int32_t *idx, int32_t *nnb) {
    int rc = check_live(c);
    if (rc != NB_OK) return rc;
    if (!n_rows || n_cap < 0) return NB_EINVAL;
    if (!c->have_ac) return NB_ESTATE;
    *n_rows = c->ac_fail_nr;
    const int64_t n = std::min<int64_t>(n_cap, c->ac_fail_nr);
    if (n > 0 && idx) NB_CUDA(c, cudaMemcpyAsync(idx, c->ac_reg_idx, sizeof(int32_t) * n, cudaMemcpyDeviceToDevice, c->stream));
    if (n > 0 && nnb) NB_CUDA(c, cudaMemcpyAsync(nnb, c->blk_nnb, sizeof(int32_t) * n, cudaMemcpyDeviceToDevice, c->stream));
    return NB_OK;
}

int nb_get_block(nb_ctx *c, int32_t n_cap, int32_t *idx_act, double *acc, double *jerk, double *pot, int32_t *nnb,
                 int32_t *nblist, int32_t *overflow) {
    int rc = check_live(c);
    if (rc != NB_OK) return rc;
    if (n_cap < 0) return NB_EINVAL;
    if (c->blk_last_two) return NB_ESTATE;      // the last block was a two-level one: its results are nb_ac_get's
    const int64_t n = std::min<int64_t>(n_cap, c->blk_last_n);      // never more rows than the caller has room for
    if (n == 0) return NB_OK;
    const cudaMemcpyKind dd = cudaMemcpyDeviceToDevice;
    if (idx_act) NB_CUDA(c, cudaMemcpyAsync(idx_act, c->blk_idx, sizeof(int32_t) * n, dd, c->stream));
    if (acc) NB_CUDA(c, cudaMemcpyAsync(acc, c->blk_out, sizeof(double) * 3 * n, dd, c->stream));
    if (jerk) NB_CUDA(c, cudaMemcpyAsync(jerk, c->blk_out + 3 * c->blk_stride, sizeof(double) * 3 * n, dd, c->stream));
    if (pot) NB_CUDA(c, cudaMemcpyAsync(pot, c->blk_out + 6 * c->blk_stride, sizeof(double) * n, dd, c->stream));
    if (nnb) NB_CUDA(c, cudaMemcpyAsync(nnb, c->blk_nnb, sizeof(int32_t) * n, dd, c->stream));
    if (overflow) NB_CUDA(c, cudaMemcpyAsync(overflow, c->blk_ovf, sizeof(int32_t) * n, dd, c->stream));
    if (nblist) {
        if (!c->blk_had_list) return NB_ESTATE;       // the step ran without h2_all: no lists were built
        NB_CUDA(c, cudaMemcpyAsync(nblist, c->blk_list, sizeof(int32_t) * n * c->cap, dd, c->stream));
    }
    return NB_OK;
}

int nb_get_state(nb_ctx *c, double *m, double *x0, double *v0, double *a0, double *j0, double *t0, double *dt) {
    int rc = check_live(c);
    if (rc != NB_OK) return rc;
    if (!m || !x0 || !v0 || !a0 || !j0 || !t0) return NB_EINVAL;
    if (!c->have_j || (dt && !c->have_steps)) return NB_ESTATE;
    export_state_kernel<<<(unsigned)((c->N + 255) / 256), 256, 0, c->stream>>>(c->N, c->Ns, c->soa, c->dtj, m, x0, v0, a0,
                                                                              j0, t0, dt);
    NB_CUDA(c, cudaGetLastError());
    c->launches += 1;
    return NB_OK;
}

int nb_set_j_offset(nb_ctx *c, int64_t j_offset) {
    int rc = check_live(c);
    if (rc != NB_OK) return rc;
    if (j_offset < 0 || j_offset + c->N > ((int64_t)1 << 31) - 1) return NB_EINVAL;
    c->j_offset = j_offset;
    return NB_OK;
}

int nb_regular_shard(nb_ctx *c, double t, int32_t n_i, const int32_t *idx_i, const double *istate, const double *h2_i,
                     double *acc, double *jerk, double *pot, int32_t *nnb, int32_t *nblist, int32_t *overflow) {
    int rc = check_live(c);
    if (rc != NB_OK) return rc;
    if (n_i < 0) return NB_EINVAL;
    if (!c->have_pred || t != c->pred_t) return NB_ESTATE;   // the shard's records must be at the same time t
    if (n_i == 0) return NB_OK;
    if (!idx_i || !istate || !h2_i || !acc || !jerk || !pot || !nnb || !nblist || !overflow) return NB_EINVAL;
    rc = materialize_pred(c);
    if (rc != NB_OK) return rc;
    const int vi = pick_variant(c, n_i);
    const Variant &v = c->var[vi];
    const int64_t n_ib = (n_i + v.iblock - 1) / v.iblock, n_i_pad = n_ib * v.iblock;
    const int64_t ntiles = c->Npad / TJ;
    const int S = pick_split(c, v, n_ib, ntiles);
    rc = ensure_partial(c, (size_t)S * 7 * n_i_pad * sizeof(double));
    if (rc != NB_OK) return rc;
    if (n_i_pad > c->ist_n) {
        NB_CUDA(c, cudaStreamSynchronize(c->stream));
        cudaFree(c->d_ist); cudaFree(c->irec); cudaFreeHost(c->h_ist);
        c->d_ist = nullptr; c->irec = nullptr; c->h_ist = nullptr; c->ist_n = 0;
        const int64_t n = std::max<int64_t>(n_i_pad, 1024) * 5 / 4;
        NB_CUDA(c, cudaMallocHost(&c->h_ist, sizeof(double) * 14 * n));
        NB_CUDA(c, cudaMalloc(&c->d_ist, sizeof(double) * 14 * n));
        NB_CUDA(c, cudaMalloc(&c->irec, sizeof(float) * RECF * n));
        c->ist_n = n;
    }
    if ((int64_t)n_i > c->cnt_n) {      // the row counters are indexed by k: a block may be larger than the shard
        NB_CUDA(c, cudaStreamSynchronize(c->stream));
        cudaFree(c->cnt); c->cnt = nullptr;
        NB_CUDA(c, cudaMalloc(&c->cnt, sizeof(int32_t) * n_i));
        NB_CUDA(c, cudaMemsetAsync(c->cnt, 0, sizeof(int32_t) * n_i, c->stream));
        c->cnt_n = n_i;
    }
    IStateSrc isrc = {};
    isrc.ist = istate;
    predict_i_kernel<false><<<(unsigned)((n_i + 255) / 256), 256, 0, c->stream>>>(n_i, (int32_t)n_i_pad, t, isrc, c->irec);
    NB_CUDA(c, cudaGetLastError());
    c->launches += 1;
    const unsigned long long *perm = nullptr;
    c->last_reordered = 0;
    if (want_reorder(c, n_i)) {
        rc = reorder_block(c, n_i, idx_i, c->irec, n_i_pad);
        if (rc != NB_OK) return rc;
        perm = c->sort_keys; c->last_reordered = 1;
    }
    rc = launch_force_range(c, vi, false, n_i, idx_i, h2_i, c->irec, perm, c->j_offset, nblist, 0, ntiles, S, 0);
    if (rc != NB_OK) return rc;
    return launch_finalize(c, n_i, n_i_pad, S, perm, acc, jerk, pot, nnb, nblist, overflow);
}

int nb_get_info(nb_ctx *c, int32_t key, int64_t *value) {
    if (!c || !value) return NB_EINVAL;
    switch (key) {
        case NB_INFO_KERNEL_LAUNCHES: *value = c->launches; break;
        case NB_INFO_LAST_JSPLIT: *value = c->last_S; break;
        case NB_INFO_LAST_IBLOCK: *value = c->last_iblock; break;
        case NB_INFO_LAST_GRID: *value = c->last_grid; break;
        case NB_INFO_SM_COUNT: *value = c->sm_count; break;
        case NB_INFO_N_PADDED: *value = c->Npad; break;
        case NB_INFO_LAST_VARIANT: *value = c->last_variant; break;
        case NB_TUNE_FORCE_JSPLIT: *value = c->force_S; break;
        case NB_TUNE_FORCE_VARIANT: *value = c->force_variant; break;
        case NB_INFO_LAST_BLOCK_N: *value = c->blk_last_two ? 0 : c->blk_last_n; break;
        case NB_TUNE_PROFILE: *value = c->profile ? 1 : 0; break;
        case NB_TUNE_STEP_CHUNKS: *value = c->step_chunks; break;
        case NB_TUNE_FUSE_PREDICT: *value = c->fuse ? 1 : 0; break;
        case NB_TUNE_LOCAL_G_MILLI: *value = (int64_t)(c->local_g * 1000.0 + 0.5); break;
        case NB_TUNE_STATS: *value = c->stats ? 1 : 0; break;
        case NB_INFO_LAST_FUSED: *value = c->last_fused; break;
        case NB_INFO_LAST_REORDERED: *value = c->last_reordered; break;
        case NB_TUNE_SPECULATE: *value = c->spec_enabled ? 1 : 0; break;
        case NB_INFO_SPEC_HITS: *value = c->spec_hits; break;
        case NB_INFO_SPEC_MISSES: *value = c->spec_misses; break;
        case NB_TUNE_REORDER_MIN: *value = c->reorder_min; break;
        case NB_TUNE_SELECT_CHUNKS: *value = c->sel_chunks ? 1 : 0; break;
        case NB_TUNE_SELECT_GRID: *value = c->sel_grid_cap; break;
        case NB_TUNE_IRR_PRED_MIN: *value = c->irr_pred_min; break;
        case NB_INFO_LOCAL_WARPS:
        case NB_INFO_TOTAL_WARPS: {
            if (!c->stats) return NB_ESTATE;
            if (c->cuda_err != cudaSuccess) return NB_ECUDA;
            unsigned int h[2] = {0, 0};
            NB_CUDA(c, cudaStreamSynchronize(c->stream));
            NB_CUDA(c, cudaMemcpy(h, c->stats, sizeof(h), cudaMemcpyDeviceToHost));
            *value = key == NB_INFO_LOCAL_WARPS ? h[0] : h[1];
            break;
        }
        case NB_INFO_FORCE_KERNEL_COUNT: *value = std::min<int64_t>(c->prof_n, nb_ctx::PROF_RING); break;
        case NB_INFO_FORCE_KERNEL_NS: {
            if (c->cuda_err != cudaSuccess) return NB_ECUDA;
            NB_CUDA(c, cudaStreamSynchronize(c->stream));
            double ns = 0.0;
            const int64_t n = std::min<int64_t>(c->prof_n, nb_ctx::PROF_RING);
            for (int64_t q = 0; q < n; ++q) {
                float ms = 0.f;
                NB_CUDA(c, cudaEventElapsedTime(&ms, c->ev0[q], c->ev1[q]));
                ns += (double)ms * 1.0e6;
            }
            *value = (int64_t)(ns + 0.5);
            break;
        }
        default:
            if (key >= NB_INFO_FORCE_KERNEL_NS_AT && key < NB_INFO_FORCE_KERNEL_NS_AT + nb_ctx::PROF_RING) {
                const int64_t q = key - NB_INFO_FORCE_KERNEL_NS_AT;       // the q-th bracketed launch
                if (q >= c->prof_n) return NB_EINVAL;
                if (c->cuda_err != cudaSuccess) return NB_ECUDA;
                NB_CUDA(c, cudaStreamSynchronize(c->stream));
                float ms = 0.f;
                NB_CUDA(c, cudaEventElapsedTime(&ms, c->ev0[q], c->ev1[q]));
                *value = (int64_t)((double)ms * 1.0e6 + 0.5);
                break;
            }
            return NB_EINVAL;
    }
    return NB_OK;
}

int nb_set_tuning(nb_ctx *c, int32_t key, int64_t value) {
    if (!c) return NB_EINVAL;
    switch (key) {
        case NB_TUNE_FORCE_JSPLIT:
            if (value < 0) return NB_EINVAL;
            c->force_S = value; break;
        case NB_TUNE_FORCE_VARIANT:
            if (value < -1 || value >= NVARIANT) return NB_EINVAL;
            c->force_variant = value; break;
        case NB_TUNE_STEP_CHUNKS:
            if (value < 0 || value > nb_ctx::MAXCHUNK) return NB_EINVAL;
            c->step_chunks = value; break;
        case NB_TUNE_FUSE_PREDICT:
            if (value != 0 && value != 1) return NB_EINVAL;
            c->fuse = value != 0;
            if (!c->fuse) return materialize_pred(c);
            break;
        case NB_TUNE_LOCAL_G_MILLI:
            if (value < 0 || value > 1000000) return NB_EINVAL;
            c->local_g = (double)value / 1000.0; break;
        case NB_TUNE_SPECULATE:
            if (value != 0 && value != 1) return NB_EINVAL;
            c->spec_enabled = value != 0; break;
        case NB_TUNE_REORDER_MIN:
            if (value < 0) return NB_EINVAL;
            c->reorder_min = value; break;
        case NB_TUNE_SELECT_CHUNKS:
            if (value != 0 && value != 1) return NB_EINVAL;
            c->sel_chunks = value != 0; break;
        case NB_TUNE_IRR_PRED_MIN:
            if (value < 0) return NB_EINVAL;
            c->irr_pred_min = value; break;
        case NB_TUNE_SELECT_GRID:
            if (value < 0) return NB_EINVAL;
            c->sel_grid_cap = value; break;
        case NB_TUNE_STATS:
            if (value != 0 && value != 1) return NB_EINVAL;
            if (value) {
                if (!c->stats) NB_CUDA(c, cudaMalloc(&c->stats, 2 * sizeof(unsigned int)));
                NB_CUDA(c, cudaMemsetAsync(c->stats, 0, 2 * sizeof(unsigned int), c->stream));
            } else if (c->stats) {
                NB_CUDA(c, cudaStreamSynchronize(c->stream));
                cudaFree(c->stats); c->stats = nullptr;
            }
            break;
        case NB_TUNE_PROFILE:
            if (value != 0 && value != 1) return NB_EINVAL;
            if (value && !c->ev0[0]) {
                for (int q = 0; q < nb_ctx::PROF_RING; ++q) {
                    NB_CUDA(c, cudaEventCreate(&c->ev0[q]));
                    NB_CUDA(c, cudaEventCreate(&c->ev1[q]));
                }
            }
            c->profile = value != 0;
            c->prof_n = 0;
            break;
        default: return NB_EINVAL;
    }
    return NB_OK;
}

int nb_plan_regular(int64_t N, int64_t n_i, int32_t sm_count, int32_t ctas_per_sm, int32_t *variant, int32_t *iblock,
                    int32_t *jsplit, int32_t *tiles_per_split) {
    if (N <= 0 || n_i <= 0 || n_i > N || sm_count <= 0 || ctas_per_sm <= 0) return NB_EINVAL;
    if (!variant || !iblock || !jsplit || !tiles_per_split) return NB_EINVAL;
    const int vi = pick_variant_pure(n_i);
    const int64_t ib = VAR_IBLOCK[vi], n_ib = (n_i + ib - 1) / ib, ntiles = (N + TJ - 1) / TJ;
    const int S = plan_split_pure((int64_t)sm_count * ctas_per_sm, VAR_OVH[vi], var_tile_us(vi), n_ib, ntiles);
    *variant = vi; *iblock = (int32_t)ib; *jsplit = S; *tiles_per_split = (int32_t)((ntiles + S - 1) / S);
    return NB_OK;
}

int nb_plan_chunks(int64_t N, int32_t chunks, int64_t *first_body, int32_t *nchunk) {
    if (N <= 0 || chunks < 0 || chunks > nb_ctx::MAXCHUNK || !first_body || !nchunk) return NB_EINVAL;
    int64_t ctile[nb_ctx::MAXCHUNK + 1];
    const int n = plan_chunks_pure((N + TJ - 1) / TJ, chunks, ctile);
    for (int q = 0; q <= n; ++q) first_body[q] = std::min<int64_t>(ctile[q] * TJ, N);
    *nchunk = n;
    return NB_OK;
}

#ifdef NBREG_TIMELINE
int nb_debug_set_timeline(void *dev_buf) {      // debug builds only: [CTA][8] uint64 stamps, NULL = off
    unsigned long long *p = static_cast<unsigned long long *>(dev_buf);
    return cudaMemcpyToSymbol(nbreg::g_timeline, &p, sizeof(p)) == cudaSuccess ? NB_OK : NB_ECUDA;
}
#endif

int nb_last_cuda_error(nb_ctx *c) { return c ? (int)c->cuda_err : 0; }

const char *nb_strerror(int code) {
    switch (code) {
        case NB_OK: return "ok";
        case NB_EINVAL: return "invalid argument";
        case NB_ESTATE: return "call out of order (set_j -> predict_all -> regular)";
        case NB_ENOMEM: return "out of device memory";
        case NB_ECUDA: return "CUDA error or no sm_100 device (see nb_last_cuda_error)";
        case NB_EOVERFLOW: return "neighbour list overflow during two-level AC stepping (shrink the radii)";
        case NB_ELIMIT: return "N exceeds NB_STATIC_MAX_N, the fixed capacity of nb_next_block_static's built-in scratch";
        default: return "unknown nbreg status";
    }
}

}  // extern "C"

// ------------------------------------------------------------------ nb_next_block_static: block selection without a context
// Who this is for: code that must pick the next block of due particles but is not allowed to allocate GPU memory at
// the point where it runs -- a plug-in living inside a host application whose memory pool already owns the whole
// device (the application hands out buffers, and a stray cudaMalloc either fails or steals from its budget), a
// real-time / in-situ analysis hook where the implicit device synchronisation of cudaMalloc and cudaFree would stall
// the simulation's other streams, or a caller running after an out-of-memory condition that still wants to know
// which bodies are due.  Such a caller cannot use nb_open (which allocates the j-state) and so cannot reach
// nb_next_block.  Here the caller brings t0, dt and the output buffers; the only working memory -- the running
// minimum and one count per 2048-body chunk -- sits in the fixed array below, which is part of the library image:
// every device that loads libnbreg reserves these 33 KB from load to exit, whether or not this call is ever made.
namespace {

constexpr int64_t SEL_STATIC_CHUNKS = NB_STATIC_MAX_N / SEL_CHUNK;                 // 8192 counts
constexpr size_t SEL_STATIC_COUNTS_OFF = 256;                                      // [0, 8): the minimum's key
constexpr size_t SEL_STATIC_BYTES = SEL_STATIC_COUNTS_OFF + sizeof(int32_t) * SEL_STATIC_CHUNKS;
static_assert(NB_STATIC_MAX_N % SEL_CHUNK == 0, "the limit is a whole number of selection chunks");

// In HOST code this name is only the host-side shadow of the symbol: it is never passed to a kernel or to
// cudaMemsetAsync.  static_scratch() asks the runtime for the array's address on the current device.
static __device__ __align__(256) unsigned char g_sel_static[SEL_STATIC_BYTES];

struct StaticScratch {
    unsigned char *base = nullptr;      // device address of g_sel_static on this device
    int sm_count = 0;
};
constexpr int STATIC_MAX_DEVICES = 64;
StaticScratch g_static_dev[STATIC_MAX_DEVICES];        // filled once per device, under g_static_mu
std::mutex g_static_mu;

// Set-up, once per device, with that device current (it is: the caller's pointers live on it).  Neither call
// allocates; cudaGetSymbolAddress may initialise the device's context and load the module if nothing of the library
// ran on it yet -- which is why the first call on a device belongs before any stream capture.
cudaError_t static_scratch(StaticScratch *out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const bool cached = dev >= 0 && dev < STATIC_MAX_DEVICES;
    std::lock_guard<std::mutex> hold(g_static_mu);
    StaticScratch s = cached ? g_static_dev[dev] : StaticScratch{};
    if (!s.base) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_sel_static);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&s.sm_count, cudaDevAttrMultiProcessorCount, dev);
        if (e == cudaSuccess && (!p || s.sm_count <= 0)) e = cudaErrorInvalidSymbol;
        if (e == cudaSuccess) {
            s.base = static_cast<unsigned char *>(p);
            if (cached) g_static_dev[dev] = s;
        }
    }
    if (e == cudaSuccess) *out = s;
    return e;
}

}  // namespace

extern "C" int nb_next_block_static(int64_t N, const double *t0, const double *dt, int32_t *idx_act,
                                    double *block, void *cuda_stream) {
    if (!t0 || !dt || !idx_act || !block || N <= 0) return NB_EINVAL;
    if (N > NB_STATIC_MAX_N) return NB_ELIMIT;           // before any CUDA call: nothing was touched
    StaticScratch s;
    if (static_scratch(&s) != cudaSuccess) return NB_ECUDA;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    unsigned long long *key = reinterpret_cast<unsigned long long *>(s.base);
    int32_t *counts = reinterpret_cast<int32_t *>(s.base + SEL_STATIC_COUNTS_OFF);
    // The array keeps what the previous call left: the key must start at "no time yet" (all ones) or the minimum
    // of an earlier call would win.  The counts need no clearing -- pass 0 writes every chunk pass 1 reads.
    if (cudaMemsetAsync(key, 0xff, sizeof(unsigned long long), stream) != cudaSuccess) return NB_ECUDA;
    const unsigned nchunk = (unsigned)((N + SEL_CHUNK - 1) / SEL_CHUNK);
    const unsigned g = (unsigned)std::min<int64_t>((N + 255) / 256, (int64_t)s.sm_count * 8);
    next_time_kernel<<<g, 256, 0, stream>>>(N, t0, dt, key);
    select_active_kernel<0><<<nchunk, 256, 0, stream>>>(N, t0, dt, key, counts, idx_act, block);
    select_active_kernel<1><<<nchunk, 256, 0, stream>>>(N, t0, dt, key, counts, idx_act, block);
    return cudaGetLastError() == cudaSuccess ? NB_OK : NB_ECUDA;
}
