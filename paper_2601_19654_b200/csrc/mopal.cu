// mopal.cu - C ABI of libmopal (include/mopal.h): context, argument checking, launch
// orchestration and the CUDA-graph step driver.  All arithmetic is in the kernels of
// pair_accel.cuh / kepler.cuh / encounters.cuh / glue.cuh.
#include <cuda_runtime.h>
#include <nvtx3/nvToolsExt.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <new>
#include <algorithm>
#include <mutex>
#include <vector>

#include "../../include/mopal.h"
#include "glue.cuh"
#include "pair_big.cuh"
#include "pair_sym.cuh"
#include "support.cuh"
#include "step_small.cuh"
#include "resolve.cuh"
#include "fixup.cuh"

using namespace mopal;

struct mo_ctx {
    int nb = 0, ld = 0, nbPad = 0, nTiles = 0, nsm = 0;
    int nbig = 0, nSrcTiles = 0;        // big bodies = gravity sources (mo_set_nbig); nbig = nb by default
    double m_star = 0, G = 0, mu = 0;
    // borrowed
    double *x = nullptr, *v = nullptr, *a = nullptr;
    const double* rcrit = nullptr;
    int* pairs = nullptr;
    long long cap = 0;
    uint8_t* flag = nullptr;
    cudaStream_t stream = nullptr;
    cudaStream_t cap_stream = nullptr;  // owned: graph capture needs a non-legacy stream
    std::vector<const void*> pair_funcs; // the O(N^2) pair kernels this context launches (graph: every other kernel node runs at high priority)
    // overlapped step: the encounter pass runs on a second (high-priority) stream beside jump + pair sum + kick,
    // reading its own copy x1, v1 of the drifted state
    bool overlap = false;
    cudaStream_t enc_stream = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    double *x1 = nullptr, *v1 = nullptr;
    // owned scratch
    double *gm = nullptr, *x0 = nullptr, *v0 = nullptr, *part = nullptr, *psumA = nullptr, *psumB = nullptr;
    unsigned* ticket = nullptr;         // two last-block counters (psumA, psumB)
    // per-step support routines
    double* gmsum = nullptr;            // sum of gm (device scalar)
    double *en_on = nullptr, *en_pair = nullptr, *en_out = nullptr;   // energy partials / result (lazy)
    double* en_host = nullptr;          // pinned, 7 doubles
    int en_npair = 0, en_split = 1;
    double res_tol = 0.0;               // mo_set_resolve: <= 0 off
    int* res_loc = nullptr;             // nb ints (lazy)
    double* res_tab = nullptr;          // extrapolation tableaux of the class-C CTAs (fallback when shared memory is short)
    int *res_label = nullptr, *res_cnp = nullptr, *res_cstart = nullptr, *res_cfill = nullptr, *res_cq = nullptr;
    int *res_clist = nullptr, *res_ctl = nullptr, *res_aux = nullptr, *res_cown = nullptr, *res_ckey = nullptr;
    double *res_dbody = nullptr, *res_dpair = nullptr;   // class D (components of more than 1023 pairs): state pools
    int *res_dbodyi = nullptr, *res_dpairi = nullptr;
    long long res_dbodyN = 0;
    int res_smemA = 0, res_smemB = 0, res_smemC = 0;
    double* fix_part = nullptr;                      // partial rows of the flagged bodies
    int *fix_list = nullptr, *fix_nf = nullptr;      // the flagged bodies, ascending (the solve beside the pair sum: fixup.cuh)
    const double* pair_x = nullptr;                  // positions the pair kernel reads (nullptr: x)
    int pair_u0 = -1, pair_u1 = -1;                  // work units of the next two-sided launch (-1: all / the rank's share)
    Gate gate = {nullptr, 0};                        // gate of the pack / pair / reduce launches being enqueued (none by default)
    int* res_mode = nullptr;                         // [0] how this step gets its accelerations (1: solve beside the pair sum,
                                                     // 0: before it), [1] what the label kernel saw (latched at the next step)
    cudaStream_t res_stream[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};   // the size classes are solved side by side
    cudaEvent_t res_fork = nullptr, res_join[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
    ResStats* res_out = nullptr;        // device
    ResStats* res_host = nullptr;       // pinned
    int hill_mode = -1;                 // mo_set_hill: -1 off
    double hill_n = 3.0;
    unsigned char* tiles = nullptr;
    EncBuf enc = {};
    DevStats* dstats = nullptr;
    DevStats* hstats = nullptr;  // pinned
    double* probe = nullptr;
    size_t ws_bytes = 0;
    // geometry
    int ipt = 1, unroll = 4, nIblk = 0, nsplit = 1, tps = 1, ctas_per_sm = 1, npsum = 0;
    // two-sided pair kernel (nb >= MO_SYM_MIN): work units and partial buffers
    int enc_split = 1;
    bool use_sym = false;
    // few gravity sources (mo_set_nbig with nbig <= MO_BIG_MAX): sources in shared memory, direct big-row encounter pass
    bool use_big = false;
    int big_ipt = 1, big_grid = 1;
    int psm_g = 8;                      // lanes per body of pair_small_kernel
    bool use_psm = false;               // nb <= PSM_MAX: pair_small_kernel (several lanes per body) instead of pack + pair + reduce
    bool use_small = false;             // nb <= SMALL_MAX: the pre-acceleration part of the step is one single-CTA kernel
    int gkernels = 0;                   // kernel launches recorded in the cached step graph
    int sym_nI = 0, sym_ch = 1, sym_nunits = 0, sym_ipt = 6;
    int4* sym_units = nullptr;
    int* sym_ustart = nullptr;
    double *sym_partI = nullptr, *sym_partJ = nullptr;
    std::vector<int4> h_units;
    std::vector<int> h_ustart;
    std::vector<long long> h_uwork;     // [nunits + 1] work before each unit, in groups of 32 columns
    int2* sym_qr = nullptr;             // [sym_nI] sharded: the column groups of each row block this rank works on
    int shard_rank = 0, shard_world = 1;   // mo_set_shard: this context computes rank's share of the pair sum (row f4)
    bool pair_ready = false;
    bool a_valid = false, snap_valid = false, box_valid = false, debug = false, use_graph = true;
    long long launches = 0;
    cudaError_t last_err = cudaSuccess;
    // graph cache (one dt)
    cudaGraphExec_t gexec = nullptr;
    double gdt = 0;
    // per-launch timing of the pair kernel
    bool timing = false;
    std::vector<cudaEvent_t> ev;  // start/stop interleaved
    size_t ev_used = 0;
};

#define CK(call)                                          \
    do {                                                  \
        cudaError_t e_ = (call);                          \
        if (e_ != cudaSuccess) {                          \
            ctx->last_err = e_;                           \
            return MO_ECUDA;                              \
        }                                                 \
    } while (0)

// NVTX range around the enqueue of a stage (header-only NVTX 3: a no-op unless a tool such as nsys is attached); the
// ranges name the stages of SURVEY.md 8(a) on a timeline of single steps (a replayed graph shows its kernels only)
struct StageRange {
    explicit StageRange(const char* name) { nvtxRangePushA(name); }
    ~StageRange() { nvtxRangePop(); }
};

static inline void shard_range(long long n, int rank, int world, long long* lo, long long* hi) {
    *lo = n * rank / world;
    *hi = n * (rank + 1) / world;
}

// The work units of the two-sided pair kernel, in launch (= dispatch) order: row blocks I ascending, each block's j tiles
// from its diagonal on in chunks of ch tiles.  All CTA slots are busy until the list runs out, and then the kernel is as
// long as the last units to finish: so the end of the list is cut finer and finer ("guided"): levels of `slots` units
// each, of .., 4, 2, 1 tiles - every level halves the spread of the slots' finishing times that the level before it left -
// and last slots / 2 tiles one GROUP of 32 columns per unit (a quarter tile: the finest piece the warp rotation works
// on).  A system with fewer tiles than two per slot (N = 4096: 272 tiles for 592 slots) is cut into groups throughout: twice
// the resident warps per SM.  Long chunks before the tail keep the units few: every unit writes a row partial of
// 24 R bytes that sym_reduce_kernel reads back (cfg3: 5599 units of at most 5 tiles -> 2700 of at most 18: half the
// DRAM traffic of the partial sums, the same kernel time; profiles/r2e_tail_and_priorities.md).
static void plan_sym_units(mo_ctx* ctx, long long tot, long long slots) {
    const int TPB = ctx->sym_ipt, ch = ctx->sym_ch;
    const long long tailQ = tot < 2 * slots ? tot : slots / 2;
    ctx->h_units.clear(); ctx->h_ustart.clear(); ctx->h_uwork.clear();
    long long seen = 0, work = 0;        // tiles before the current one; groups before the current unit
    for (int I = 0; I < ctx->sym_nI; ++I) {
        ctx->h_ustart.push_back((int)ctx->h_units.size());
        int t = I * TPB;
        while (t < ctx->nTiles) {
            const long long left = tot - seen;                 // tiles from here to the end of the list
            if (left <= tailQ) {
                for (int g = 0; g < TJ / 32; ++g) {
                    ctx->h_uwork.push_back(work); work += 1;
                    ctx->h_units.push_back(make_int4(I, t, t + 1, g | (g + 1) << 8));
                }
                t += 1; seen += 1;
                continue;
            }
            // (the first tenth of the work in units of two tiles: in the resolving step it is launched on its own, beside
            // the encounter pass, and the encounter solve's CTAs - whole SMs - can only start when its CTAs have left:
            // cfg3 with resolution 3.45 ms per step with units of 4 tiles there, 3.39 with 2, 3.37 with 1)
            int n = seen < tot / 10 && ch > 2 ? 2 : ch;
            long long lo = tailQ;                               // where the next finer level begins
            for (int m = 1; m < ch; m *= 2) {
                if (left <= lo + slots * m) { n = m < n ? m : n; break; }
                lo += slots * m;
            }
            if (n > ctx->nTiles - t) n = ctx->nTiles - t;
            if (left - n < lo) n = (int)(left - lo);            // the chunk ends where the finer tail begins
            ctx->h_uwork.push_back(work); work += (long long)n * (TJ / 32);
            ctx->h_units.push_back(make_int4(I, t, t + n, (TJ / 32) << 8));
            t += n; seen += n;
        }
    }
    ctx->h_ustart.push_back((int)ctx->h_units.size());
    ctx->h_uwork.push_back(work);
    ctx->sym_nunits = (int)ctx->h_units.size();
}

// this rank's run of the work units: equal shares of the WORK (the units differ in length)
static void sym_shard_units(const mo_ctx* ctx, long long* u0, long long* u1) {
    *u0 = 0; *u1 = ctx->sym_nunits;
    if (ctx->shard_world <= 1) return;
    const long long W = ctx->h_uwork.back();
    long long wlo, whi;
    shard_range(W, ctx->shard_rank, ctx->shard_world, &wlo, &whi);
    auto first_at = [&](long long w) { return (long long)(std::lower_bound(ctx->h_uwork.begin(), ctx->h_uwork.end() - 1, w) - ctx->h_uwork.begin()); };
    *u0 = first_at(wlo);
    *u1 = ctx->shard_rank == ctx->shard_world - 1 ? ctx->sym_nunits : first_at(whi);
}

// sharded: the run of column groups of every row block (counted from the block's diagonal) that this rank's units cover
static cudaError_t sym_fill_qr(mo_ctx* ctx) {
    long long u0, u1;
    sym_shard_units(ctx, &u0, &u1);
    std::vector<int2> qr((size_t)ctx->sym_nI, make_int2(0, 0));
    const int G = TJ / 32;
    for (long long u = u0; u < u1; ++u) {
        const int4 un = ctx->h_units[(size_t)u];
        const int first = (un.y - un.x * ctx->sym_ipt) * G + (un.w & 0xff);
        const int end = (un.z - 1 - un.x * ctx->sym_ipt) * G + (un.w >> 8);
        int2& q = qr[(size_t)un.x];
        if (q.y == q.x) q = make_int2(first, end); else q.y = end;      // the units of a block follow one another
    }
    cudaError_t e = cudaMemcpyAsync(ctx->sym_qr, qr.data(), qr.size() * sizeof(int2), cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);       // pageable source
    return e;
}

static inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

static mo_status post_launch(mo_ctx* ctx, int n = 1) {
    ctx->launches += n;
    CK(cudaGetLastError());
    if (ctx->debug) CK(cudaStreamSynchronize(ctx->stream));
    return MO_OK;
}

template <typename T>
static cudaError_t dalloc(mo_ctx* ctx, T** p, size_t n) {
    size_t bytes = n * sizeof(T);
    if (bytes == 0) bytes = 16;
    cudaError_t e = cudaMalloc(reinterpret_cast<void**>(p), bytes);
    if (e == cudaSuccess) ctx->ws_bytes += bytes;
    return e;
}

typedef void (*pair_kernel_t)(AccelParams);
static pair_kernel_t pick_pair_kernel(int ipt, int unroll) {
    if (ipt == 1) return unroll == 2 ? pair_accel_kernel<1, 2> : pair_accel_kernel<1, 4>;
    return unroll == 4 ? pair_accel_kernel<2, 4> : pair_accel_kernel<2, 2>;
}

// Environment switches (read at mo_create / mo_set_nbig; documented in include/mopal.h): MO_DEBUG, and the five the
// tests use to force a kernel that the size alone would not select - MO_PSM, MO_SYM, MO_SYM_CH, MO_SYM_IPT, MO_SMALL, MO_SMALL_MAX.
static int env_int(const char* name, int dflt) {
    const char* s = getenv(name);
    return (s && *s) ? atoi(s) : dflt;
}

typedef void (*sym_kernel_t)(SymParams);
static sym_kernel_t pick_sym_kernel(int ipt) {
    return ipt == 2 ? pair_sym_kernel<2> : ipt == 3 ? pair_sym_kernel<3> : pair_sym_kernel<6>;
}
static constexpr int SYM_MIN = 2561;   // right above the lane-split kernel's range

typedef void (*big_kernel_t)(BigParams);
static big_kernel_t pick_big_kernel(int ipt, bool kick) {
    if (ipt == 4 && false) return kick ? pair_big_kernel<4, 2, true> : pair_big_kernel<4, 2, false>;
    if (ipt == 4) return kick ? pair_big_kernel<4, 1, true> : pair_big_kernel<4, 1, false>;
    if (ipt == 2) return kick ? pair_big_kernel<2, 2, true> : pair_big_kernel<2, 2, false>;
    return kick ? pair_big_kernel<1, 4, true> : pair_big_kernel<1, 4, false>;
}

// j-split count: minimise (waves) x (tiles per CTA + start-up), see DESIGN.md section 5
static void choose_geometry(mo_ctx* ctx) {
    const int nb = ctx->nb;
    ctx->ipt = nb >= 8192 ? 2 : 1;
    if (ctx->ipt != 1 && ctx->ipt != 2) ctx->ipt = 1;
    ctx->unroll = ctx->ipt == 2 ? 2 : 4;
    if (ctx->unroll != 2 && ctx->unroll != 4) ctx->unroll = 4;
    const int rows = CONSUMER_THREADS * ctx->ipt;
    ctx->nIblk = (nb + rows - 1) / rows;
    int occ = 1;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, pick_pair_kernel(ctx->ipt, ctx->unroll), CTA_THREADS, 0);
    if (occ < 1) occ = 1;
    ctx->ctas_per_sm = occ;
    const long long slots = (long long)ctx->nsm * occ;
    const int nST = ctx->nSrcTiles;       // j tiles that hold a gravity source
    const int smax = nST < 48 ? nST : 48;
    double best = 1e300;
    int bestS = 1;
    for (int S = 1; S <= smax; ++S) {
        const int tps = (nST + S - 1) / S;
        const int Se = (nST + tps - 1) / tps;
        const long long ctas = (long long)ctx->nIblk * Se;
        const long long waves = (ctas + slots - 1) / slots;
        const double cost = (double)waves * (tps + 1.5);
        if (cost < best * (1.0 - 1e-9)) { best = cost; bestS = Se; }
    }
    ctx->tps = (nST + bestS - 1) / bestS;
    ctx->nsplit = (nST + ctx->tps - 1) / ctx->tps;
    // encounter find: column tiles of a row tile are dealt round-robin to enc_split CTAs
    // (up to 8 for the large systems, whose dense rows overlap many tiles; a mid-size system's few row tiles are split
    // further, down to two column tiles per CTA: about four CTAs per SM, and a short chain of gates per thread)
    ctx->enc_split = ctx->nTiles / 8;
    if (ctx->enc_split < 1) ctx->enc_split = 1;
    if (ctx->enc_split > 8) ctx->enc_split = 8;
    {
        // (without the spatial ordering, up to 40 tiles: one column tile per CTA - the exact tests of a giant's row, which
        // passes the gate against thousands of bodies, are the long pole of the pass)
        int want = 4 * ctx->nsm / (ctx->nTiles > 0 ? ctx->nTiles : 1), most = ctx->nTiles <= ENC_UNSORTED_TILES ? ctx->nTiles : ctx->nTiles / 2;
        if (ctx->nTiles <= ENC_UNSORTED_TILES) want = 32;
        if (want > 32) want = 32;
        if (want > most) want = most;
        if (want > ctx->enc_split) ctx->enc_split = want;
    }
    // two-sided kernel for large nb: units = (row block, chunk of sym_ch j tiles from the diagonal on)
    ctx->use_small = nb <= env_int("MO_SMALL_MAX", 320) && nb <= SMALL_MAX && env_int("MO_SMALL", 1) != 0;
    // measured (profiles/r1g_path_selection.md): single-CTA front end up to ~320 bodies, lane-split pair kernel up to
    // ~2500, tiled one-sided kernel up to 8191, two-sided kernel above
    ctx->use_psm = nb <= 2560 && nb <= PSM_MAX && env_int("MO_PSM", 1) != 0;
    ctx->psm_g = 8;
    if (ctx->psm_g != 2 && ctx->psm_g != 4 && ctx->psm_g != 8) ctx->psm_g = 8;
    ctx->use_big = !ctx->use_psm && ctx->nbig < nb && ctx->nbig <= 4096;
    if (ctx->use_big) {
        // bodies per thread: as many as still leave about two waves of CTAs
        const long long want = 2LL * ctx->nsm * BIG_THREADS;
        ctx->big_ipt = nb >= 2 * want ? 2 : 1;   // 4 measured no faster (register-bound occupancy)
        if (ctx->big_ipt != 1 && ctx->big_ipt != 2 && ctx->big_ipt != 4) ctx->big_ipt = 1;
        ctx->ipt = ctx->big_ipt; ctx->nsplit = 1; ctx->tps = ctx->nSrcTiles;
        ctx->nIblk = (nb + BIG_THREADS * ctx->big_ipt - 1) / (BIG_THREADS * ctx->big_ipt);
        int occb = 1;
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occb, pick_big_kernel(ctx->big_ipt, true), BIG_THREADS, 0);
        if (occb < 1) occb = 1;
        ctx->ctas_per_sm = occb;
        ctx->big_grid = ctx->nIblk < ctx->nsm * occb ? ctx->nIblk : ctx->nsm * occb;   // persistent: CTAs walk over i blocks
    }
    // two-sided kernel: from SYM_MIN bodies on (below, the lane-split kernel's single launch wins)
    ctx->use_sym = !ctx->use_psm && ctx->nbig == nb && env_int("MO_SYM", nb >= SYM_MIN ? 1 : 0) != 0;
    if (ctx->use_sym) {
        // bodies per lane: the triangle of a mid-size system in enough, short enough units for the SMs
        ctx->sym_ipt = env_int("MO_SYM_IPT", nb >= 20000 ? 6 : nb >= 7000 ? 3 : 2);   // measured: profiles/r2c_path_selection.md, r2e_tail_and_priorities.md
        if (ctx->sym_ipt != 2 && ctx->sym_ipt != 3 && ctx->sym_ipt != 6) ctx->sym_ipt = 6;
        const int R = sym_rows(ctx->sym_ipt), TPB = ctx->sym_ipt;
        int occs = 1;
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occs, pick_sym_kernel(ctx->sym_ipt), SYM_THREADS, 0);
        if (occs < 1) occs = 1;
        const long long sslots = (long long)ctx->nsm * occs;
        ctx->sym_nI = (ctx->nbPad + R - 1) / R;
        long long tot = 0;
        for (int I = 0; I < ctx->sym_nI; ++I) tot += ctx->nTiles - I * TPB;
        long long ch = (tot + 4 * sslots - 1) / (4 * sslots);     // about four waves of long units before the guided tail (plan_sym_units)
        if (ch < 4) ch = 4;
        if (ch > 24) ch = 24;
        ctx->sym_ch = env_int("MO_SYM_CH", (int)ch);
        if (ctx->sym_ch > 64) ctx->sym_ch = 64;
        if (ctx->sym_ch < 1) ctx->sym_ch = 1;
        plan_sym_units(ctx, tot, sslots);
        ctx->ipt = ctx->sym_ipt; ctx->ctas_per_sm = occs; ctx->nsplit = 1;
    }
}

extern "C" const char* mo_strerror(mo_status s) {
    switch (s) {
        case MO_OK: return "ok";
        case MO_EINVAL: return "invalid argument";
        case MO_ENOMEM: return "out of device memory";
        case MO_ECUDA: return "CUDA error or no CUDA device";
        case MO_EOVERFLOW: return "more encounter pairs than cap";
        case MO_ENOCONV: return "Kepler solve failed for at least one body";
        case MO_ERESOLVE: return "at least one encounter component was not resolved";
        case MO_ELIMIT: return "size beyond the fixed maximum of a no-allocation entry point (mo_accel_static_max_nb)";
    }
    return "unknown status";
}

extern "C" const char* mo_version(void) { return "libmopal 0.1 (sm_100a)"; }

extern "C" void mo_destroy(mo_ctx* ctx) {
    if (!ctx) return;
    if (ctx->gexec) cudaGraphExecDestroy(ctx->gexec);
    if (ctx->cap_stream) cudaStreamDestroy(ctx->cap_stream);
    if (ctx->enc_stream) cudaStreamDestroy(ctx->enc_stream);
    if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
    if (ctx->ev_join) cudaEventDestroy(ctx->ev_join);
    cudaFree(ctx->x1); cudaFree(ctx->v1);
    for (cudaEvent_t e : ctx->ev) cudaEventDestroy(e);
    cudaFree(ctx->gm); cudaFree(ctx->x0); cudaFree(ctx->v0); cudaFree(ctx->part);
    cudaFree(ctx->psumA); cudaFree(ctx->psumB); cudaFree(ctx->ticket);
    cudaFree(ctx->res_loc); cudaFree(ctx->res_out); cudaFree(ctx->res_tab); cudaFree(ctx->res_label);
    cudaFree(ctx->res_cnp); cudaFree(ctx->res_cstart); cudaFree(ctx->res_cfill); cudaFree(ctx->res_cq); cudaFree(ctx->res_clist); cudaFree(ctx->res_ctl); cudaFree(ctx->res_aux); cudaFree(ctx->res_cown); cudaFree(ctx->res_ckey); cudaFree(ctx->fix_list); cudaFree(ctx->fix_nf); cudaFree(ctx->fix_part); cudaFree(ctx->res_mode);
    cudaFree(ctx->res_dbody); cudaFree(ctx->res_dpair); cudaFree(ctx->res_dbodyi); cudaFree(ctx->res_dpairi);
    if (ctx->res_host) cudaFreeHost(ctx->res_host);
    for (int k = 0; k < 5; ++k) { if (ctx->res_stream[k]) cudaStreamDestroy(ctx->res_stream[k]); if (ctx->res_join[k]) cudaEventDestroy(ctx->res_join[k]); }
    if (ctx->res_fork) cudaEventDestroy(ctx->res_fork);
    cudaFree(ctx->gmsum); cudaFree(ctx->en_on); cudaFree(ctx->en_pair); cudaFree(ctx->en_out);
    if (ctx->en_host) cudaFreeHost(ctx->en_host); cudaFree(ctx->tiles);
    cudaFree(ctx->sym_units); cudaFree(ctx->sym_ustart); cudaFree(ctx->sym_partI); cudaFree(ctx->sym_partJ); cudaFree(ctx->sym_qr);
    cudaFree(ctx->enc.box); cudaFree(ctx->enc.boxf); cudaFree(ctx->enc.rowcnt); cudaFree(ctx->enc.rowfill);
    cudaFree(ctx->enc.rowoff); cudaFree(ctx->enc.hits); cudaFree(ctx->enc.tmpj); cudaFree(ctx->enc.nhit);
    cudaFree(ctx->enc.ovf_now); cudaFree(ctx->dstats); cudaFree(ctx->probe);
    cudaFree(ctx->enc.bpart); cudaFree(ctx->enc.cellcnt); cudaFree(ctx->enc.cellfill); cudaFree(ctx->enc.key);
    cudaFree(ctx->enc.perm); cudaFree(ctx->enc.sboxf); cudaFree(ctx->enc.tbox); cudaFree(ctx->enc.tilecnt);
    cudaFree(ctx->enc.tbig); cudaFree(ctx->enc.nlong); cudaFree(ctx->enc.longrows);
    if (ctx->hstats) cudaFreeHost(ctx->hstats);
    delete ctx;
}

extern "C" mo_status mo_create(mo_ctx** out, int32_t nb, int32_t ld, double m_star, double G, const double* mass,
                               double* x, double* v, double* a, const double* rcrit, int32_t* pairs, int64_t cap,
                               uint8_t* flag, void* cuda_stream) {
    if (!out) return MO_EINVAL;
    *out = nullptr;
    if (nb < 1 || ld < nb || (ld & 3) || !mass || !x || !v || !a || !rcrit || !flag || cap < 0 || (cap > 0 && !pairs))
        return MO_EINVAL;
    if (!(m_star > 0.0) || !(G > 0.0) || !isfinite(m_star) || !isfinite(G)) return MO_EINVAL;
    if (!aligned16(x) || !aligned16(v) || !aligned16(a) || !aligned16(mass) || !aligned16(rcrit)) return MO_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return MO_ECUDA; }
    mo_ctx* ctx = new (std::nothrow) mo_ctx();
    if (!ctx) return MO_ENOMEM;
    ctx->nb = nb; ctx->ld = ld; ctx->m_star = m_star; ctx->G = G; ctx->mu = G * m_star;
    ctx->x = x; ctx->v = v; ctx->a = a; ctx->rcrit = rcrit; ctx->pairs = pairs; ctx->cap = cap; ctx->flag = flag;
    ctx->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    ctx->debug = env_int("MO_DEBUG", 0) != 0;
    ctx->use_graph = true;
    ctx->nTiles = (nb + TJ - 1) / TJ;
    ctx->nbPad = ctx->nTiles * TJ;
    ctx->nbig = nb; ctx->nSrcTiles = ctx->nTiles;
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
        cudaGetLastError(); delete ctx; return MO_ECUDA;
    }
    if (prop.major < 10) { delete ctx; return MO_ECUDA; }  // sm_100a code only
    ctx->nsm = prop.multiProcessorCount;
    choose_geometry(ctx);
    ctx->npsum = (ctx->nbPad + ON_BLOCK - 1) / ON_BLOCK;
    cudaError_t e = cudaSuccess;
    const size_t pl = 3 * (size_t)ld;
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->gm, (size_t)nb);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->x0, pl);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->v0, pl);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->psumA, 3 * (size_t)ctx->npsum + 3);   // partials + their sum
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->psumB, 3 * (size_t)ctx->npsum + 3);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->gmsum, 1);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->ticket, 2);
    if (e == cudaSuccess) e = cudaMemsetAsync(ctx->ticket, 0, 2 * sizeof(unsigned), ctx->stream);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->tiles, (size_t)ctx->nTiles * SYM_TILE_BYTES);   // the larger of the two tile layouts
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->enc.box, (size_t)ctx->nbPad);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->enc.boxf, (size_t)ctx->nbPad);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->enc.rowcnt, (size_t)ctx->nbPad);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->enc.rowfill, (size_t)ctx->nbPad);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->enc.rowoff, (size_t)ctx->nbPad);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->enc.hits, (size_t)cap);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->enc.tmpj, (size_t)cap);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->enc.nhit, 1);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->enc.ovf_now, 1);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->enc.bpart, (size_t)ctx->npsum);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->enc.cellcnt, (size_t)ENC_NCELL);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->enc.cellfill, (size_t)ENC_NCELL);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->enc.key, (size_t)ctx->nbPad);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->enc.perm, (size_t)ctx->nbPad);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->enc.sboxf, (size_t)ctx->nbPad);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->enc.tbox, (size_t)ctx->nTiles);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->enc.tilecnt, (size_t)ctx->nTiles);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->enc.tbig, (size_t)ctx->nTiles);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->enc.nlong, 1);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->enc.longrows, (size_t)(cap / ENC_RANK_LONG + 1));
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->dstats, 1);
    if (e == cudaSuccess) e = cudaMallocHost(reinterpret_cast<void**>(&ctx->hstats), sizeof(DevStats));
    if (e != cudaSuccess) {
        cudaGetLastError();
        mo_destroy(ctx);
        return e == cudaErrorMemoryAllocation ? MO_ENOMEM : MO_ECUDA;
    }
    e = cudaMemsetAsync(ctx->dstats, 0, sizeof(DevStats), ctx->stream);
    if (e == cudaSuccess) {
        gm_kernel<<<(nb + 255) / 256, 256, 0, ctx->stream>>>(mass, G, nb, ctx->gm);
        gmsum_kernel<<<1, 1024, 0, ctx->stream>>>(ctx->gm, nb, ctx->gmsum);
        ctx->launches += 2;
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);  // `mass` is borrowed only during the call
    if (e != cudaSuccess) { mo_destroy(ctx); return MO_ECUDA; }
    *out = ctx;
    return MO_OK;
}

// ---- stage launchers -------------------------------------------------------------------------
// partial-sum buffers of the pair kernels: allocated at the first mo_accel / mo_step, so that a context
// used only for mo_drift / mo_encounters (e.g. a bandwidth sweep at 2^24 bodies) does not pay for them
static mo_status ensure_pair_scratch(mo_ctx* ctx) {
    if (ctx->pair_ready) return MO_OK;
    cudaError_t e = cudaSuccess;
    ctx->overlap = !ctx->use_small;
    if (ctx->overlap && !ctx->enc_stream) {
        int lo = 0, hi = 0;
        cudaDeviceGetStreamPriorityRange(&lo, &hi);
        e = cudaStreamCreateWithPriority(&ctx->enc_stream, cudaStreamNonBlocking, hi);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_join, cudaEventDisableTiming);
        if (e == cudaSuccess) e = dalloc(ctx, &ctx->x1, 3 * (size_t)ctx->ld);
        if (e == cudaSuccess) e = dalloc(ctx, &ctx->v1, 3 * (size_t)ctx->ld);
    }
    const size_t pl = 3 * (size_t)ctx->ld;
    if (e == cudaSuccess && !ctx->use_sym && !ctx->use_big && !ctx->use_psm) e = dalloc(ctx, &ctx->part, pl * (size_t)ctx->nsplit);
    if (ctx->use_sym) {
        if (e == cudaSuccess) e = dalloc(ctx, &ctx->sym_units, (size_t)ctx->sym_nunits);
        if (e == cudaSuccess) e = dalloc(ctx, &ctx->sym_ustart, ctx->h_ustart.size());
        if (e == cudaSuccess) e = dalloc(ctx, &ctx->sym_partI, (size_t)ctx->sym_nunits * 3 * sym_rows(ctx->sym_ipt));
        if (e == cudaSuccess) e = dalloc(ctx, &ctx->sym_partJ, (size_t)symJ_off(ctx->sym_nI, ctx->nbPad, sym_rows(ctx->sym_ipt)));
        if (e == cudaSuccess) e = cudaMemcpyAsync(ctx->sym_units, ctx->h_units.data(), ctx->h_units.size() * sizeof(int4), cudaMemcpyHostToDevice, ctx->stream);
        if (e == cudaSuccess) e = cudaMemcpyAsync(ctx->sym_ustart, ctx->h_ustart.data(), ctx->h_ustart.size() * sizeof(int), cudaMemcpyHostToDevice, ctx->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);   // pageable source vectors
        if (e == cudaSuccess) e = dalloc(ctx, &ctx->sym_qr, (size_t)ctx->sym_nI);
        if (e == cudaSuccess) e = sym_fill_qr(ctx);
    }
    if (e != cudaSuccess) {
        cudaGetLastError();
        ctx->last_err = e;
        ctx->overlap = false;      // never run the forked step on half-made streams / copies
        return e == cudaErrorMemoryAllocation ? MO_ENOMEM : MO_ECUDA;
    }
    ctx->pair_ready = true;
    return MO_OK;
}

static void note_pair_func(mo_ctx* ctx, const void* f) {
    if (std::find(ctx->pair_funcs.begin(), ctx->pair_funcs.end(), f) == ctx->pair_funcs.end()) ctx->pair_funcs.push_back(f);
}

// The recorded step replays with the priorities of its nodes (cudaGraphInstantiateFlagUseNodePriority; without the flag
// every node runs at the priority of the stream the graph is launched into): the pair kernel, whose CTAs take every
// slot of the GPU for the length of the step, at the lowest, every other kernel - the encounter branch and the
// encounter solve beside it, chains of short dependent kernels - at the highest, so that a slot a pair CTA leaves goes
// to them first.  (Measured at N = 16,384: without it the encounter branch only got onto the GPU when the pair kernel's
// grid had been handed out, and the replayed step was as long as with no overlap at all.)
static cudaError_t set_node_priorities(mo_ctx* ctx, cudaGraph_t g) {
    int lo = 0, hi = 0;
    cudaError_t e = cudaDeviceGetStreamPriorityRange(&lo, &hi);
    size_t n = 0;
    if (e == cudaSuccess) e = cudaGraphGetNodes(g, nullptr, &n);
    if (e != cudaSuccess || n == 0) return e;
    std::vector<cudaGraphNode_t> nodes(n);
    e = cudaGraphGetNodes(g, nodes.data(), &n);
    for (size_t k = 0; k < n && e == cudaSuccess; ++k) {
        cudaGraphNodeType ty;
        e = cudaGraphNodeGetType(nodes[k], &ty);
        if (e != cudaSuccess || ty != cudaGraphNodeTypeKernel) continue;
        cudaKernelNodeParams kp;
        e = cudaGraphKernelNodeGetParams(nodes[k], &kp);
        if (e != cudaSuccess) break;
        const bool pair = std::find(ctx->pair_funcs.begin(), ctx->pair_funcs.end(), (const void*)kp.func) != ctx->pair_funcs.end();
        cudaLaunchAttributeValue v;
        memset(&v, 0, sizeof v);
        v.priority = pair ? lo : hi;
        e = cudaGraphKernelNodeSetAttribute(nodes[k], cudaLaunchAttributePriority, &v);
    }
    return e;
}

static mo_status launch_pair(mo_ctx* ctx, bool kick = false, double hk = 0.0) {
    AccelParams p;
    p.tiles = ctx->tiles; p.x = ctx->x; p.rcrit = ctx->rcrit; p.part = ctx->part;
    p.nb = ctx->nb; p.ld = ctx->ld; p.nTiles = ctx->nSrcTiles; p.tps = ctx->tps;
    dim3 grid(ctx->nIblk, ctx->nsplit);
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    const bool timed = ctx->timing && !ctx->gate.flag;    // a gated launch may be a no-op: not a kernel time
    if (timed) {
        if (ctx->ev_used + 2 > ctx->ev.size()) {
            cudaEvent_t a, b;
            CK(cudaEventCreate(&a)); CK(cudaEventCreate(&b));
            ctx->ev.push_back(a); ctx->ev.push_back(b);
        }
        e0 = ctx->ev[ctx->ev_used]; e1 = ctx->ev[ctx->ev_used + 1];
        ctx->ev_used += 2;
        CK(cudaEventRecord(e0, ctx->stream));
    }
    if (ctx->use_psm) {
        BigParams bp;
        bp.x = ctx->x; bp.gm = ctx->gm; bp.rcrit = ctx->rcrit; bp.a = ctx->a; bp.v = ctx->v;
        bp.nb = ctx->nb; bp.nbig = ctx->nbig; bp.ld = ctx->ld; bp.hk = hk; bp.blk0 = 0; bp.blk1 = 0;
        const int G = ctx->psm_g, per = PSM_THREADS / G;
        const int grid = (ctx->nb + per - 1) / per;
        auto k = G == 8 ? (kick ? pair_small_kernel<8, true> : pair_small_kernel<8, false>)
               : G == 4 ? (kick ? pair_small_kernel<4, true> : pair_small_kernel<4, false>)
                        : (kick ? pair_small_kernel<2, true> : pair_small_kernel<2, false>);
        note_pair_func(ctx, (const void*)k);
        k<<<grid, PSM_THREADS, 0, ctx->stream>>>(bp);
    } else if (ctx->use_big) {
        BigParams bp;
        bp.x = ctx->x; bp.gm = ctx->gm; bp.rcrit = ctx->rcrit; bp.a = ctx->a; bp.v = ctx->v;
        bp.nb = ctx->nb; bp.nbig = ctx->nbig; bp.ld = ctx->ld; bp.hk = hk; bp.blk0 = 0; bp.blk1 = 0;
        int grid = ctx->big_grid;
        if (ctx->shard_world > 1) {       // this rank's blocks of bodies i; the other rows of a stay 0 (the caller sums over the ranks)
            long long lo, hi;
            shard_range(ctx->nIblk, ctx->shard_rank, ctx->shard_world, &lo, &hi);
            bp.blk0 = (int)lo; bp.blk1 = (int)hi;
            CK(cudaMemsetAsync(ctx->a, 0, 3 * (size_t)ctx->ld * sizeof(double), ctx->stream));
            grid = hi - lo < grid ? (int)(hi - lo) : grid;
        }
        if (grid > 0 && (ctx->shard_world == 1 || bp.blk1 > bp.blk0))
            { note_pair_func(ctx, (const void*)pick_big_kernel(ctx->big_ipt, kick)); pick_big_kernel(ctx->big_ipt, kick)<<<grid, BIG_THREADS, 0, ctx->stream>>>(bp); }
    } else if (ctx->use_sym) {
        SymParams sp;
        sp.tiles = ctx->tiles; sp.x = ctx->pair_x ? ctx->pair_x : ctx->x; sp.gm = ctx->gm; sp.rcrit = ctx->rcrit; sp.units = ctx->sym_units;
        sp.partI = ctx->sym_partI; sp.partJ = ctx->sym_partJ; sp.nb = ctx->nb; sp.ld = ctx->ld; sp.nbPad = ctx->nbPad;
        long long u0, u1;
        sym_shard_units(ctx, &u0, &u1);
        if (ctx->pair_u0 >= 0) { u0 = ctx->pair_u0; u1 = ctx->pair_u1; }
        sp.unit0 = (int)u0; sp.gate = ctx->gate;
        note_pair_func(ctx, (const void*)pick_sym_kernel(ctx->sym_ipt));
        if (u1 > u0) pick_sym_kernel(ctx->sym_ipt)<<<(int)(u1 - u0), SYM_THREADS, 0, ctx->stream>>>(sp);
    } else {
        note_pair_func(ctx, (const void*)pick_pair_kernel(ctx->ipt, ctx->unroll));
        pick_pair_kernel(ctx->ipt, ctx->unroll)<<<grid, CTA_THREADS, 0, ctx->stream>>>(p);
    }
    if (timed) CK(cudaEventRecord(e1, ctx->stream));
    return post_launch(ctx);
}

// a <- accel(x), optionally preceded by the jump (psumB) and followed by the kick
static mo_status enqueue_accel(mo_ctx* ctx, bool jump, double hj, bool kick, double hk) {
    StageRange nv("mopal: jump + pair accelerations + kick (a4, a1, a2, a3)");
    if (ctx->shard_world > 1) kick = false;      // a is this rank's share: the kick follows the caller's sum over the ranks (mo_step_end)
    const double hjm = jump ? hj / ctx->mu : 0.0;
    const double* ps = jump ? ctx->psumB : nullptr;
    const int nps = jump ? ctx->npsum : 0;
    if (ctx->use_big || ctx->use_psm) {
        // the jump still moves every body (pack_kernel also refreshes the few source tiles, unused here);
        // pair_big_kernel reads the sources from x, writes a itself and applies the closing kick
        if (jump) {
            pack_kernel<true, false><<<ctx->nTiles, TJ, 0, ctx->stream>>>(ctx->x, ctx->gm, ctx->rcrit, ctx->nb, ctx->nbig, ctx->ld,
                                                                        ctx->tiles, ps, nps, hjm, ctx->gate);
            mo_status s = post_launch(ctx);
            if (s != MO_OK) return s;
        }
        return launch_pair(ctx, kick, hk);
    }
    auto pk = jump ? (ctx->use_sym ? pack_kernel<true, true> : pack_kernel<true, false>)
                   : (ctx->use_sym ? pack_kernel<false, true> : pack_kernel<false, false>);
    pk<<<jump ? ctx->nTiles : ctx->nSrcTiles, TJ, 0, ctx->stream>>>(ctx->x, ctx->gm, ctx->rcrit, ctx->nb, ctx->nbig, ctx->ld,
                                                                    ctx->tiles, ps, nps, hjm, ctx->gate);
    mo_status s = post_launch(ctx);
    if (s != MO_OK) return s;
    s = launch_pair(ctx);
    if (s != MO_OK) return s;
    const int nblk = (ctx->nb + ON_BLOCK - 1) / ON_BLOCK;
    if (ctx->use_sym) {
        const bool shd = ctx->shard_world > 1;
        auto rk = kick ? sym_reduce_kernel<true, false> : shd ? sym_reduce_kernel<false, true> : sym_reduce_kernel<false, false>;
        long long u0, u1;
        sym_shard_units(ctx, &u0, &u1);
        rk<<<dim3((ctx->nb + 31) / 32, 3), RED_THREADS, 0, ctx->stream>>>(ctx->sym_partI, ctx->sym_partJ, ctx->sym_ustart, ctx->nb, ctx->ld, ctx->nbPad,
                                               ctx->a, kick ? ctx->v : nullptr, kick ? hk : 0.0, (int)u0, (int)u1, ctx->sym_qr, sym_rows(ctx->sym_ipt), ctx->gate);
    } else if (kick)
        accel_reduce_kernel<true><<<nblk, ON_BLOCK, 0, ctx->stream>>>(ctx->part, ctx->nsplit, ctx->nb, ctx->ld, ctx->a, ctx->v, hk);
    else
        accel_reduce_kernel<false><<<nblk, ON_BLOCK, 0, ctx->stream>>>(ctx->part, ctx->nsplit, ctx->nb, ctx->ld, ctx->a, nullptr, 0.0);
    return post_launch(ctx);
}

static EncState enc_state(const mo_ctx* ctx, const double* x0, const double* v0, double h) {
    EncState s;
    s.x0 = x0; s.v0 = v0; s.x1 = ctx->x; s.v1 = ctx->v; s.rcrit = ctx->rcrit;
    s.nb = ctx->nb; s.ld = ctx->ld; s.nbig = ctx->nbig; s.h = h;
    return s;
}

// find + scan + place (+ overflow fallback) on boxes already in ctx->enc (counters already zeroed)
static mo_status enqueue_pairs(mo_ctx* ctx, const EncState& es, int step_inc) {
    StageRange nv("mopal: encounter pairs (a8)");
    EncFindParams fp;
    fp.s = es; fp.e = ctx->enc; fp.cap = ctx->cap; fp.nTiles = ctx->nTiles;
    // up to 40 tiles (N <= 5120) every pair of tiles is gated, in body order: that costs less than the three ordering
    // kernels in a chain of dependent launches this short (at N = 4096 the chain, not the pair sum, was the step: 61 ->
    // 50.5 us; equal at N = 6000, and at N = 8192 the ordering wins by 15 us)
    fp.unsorted = ctx->nTiles <= ENC_UNSORTED_TILES ? 1 : 0;
    mo_status s;
    if (ctx->use_big) {
        // few big bodies: the nbig x nb rectangle of gates directly, in body order
        const int per = BIGF_THREADS * BIGF_JPT;
        enc_bigfind_kernel<<<(ctx->nb + per - 1) / per, BIGF_THREADS, 0, ctx->stream>>>(fp);
        s = post_launch(ctx);
        if (s != MO_OK) return s;
    } else if (fp.unsorted) {
        enc_find_kernel<<<dim3(ctx->nTiles, ctx->enc_split), CTA_THREADS, 0, ctx->stream>>>(fp);
        s = post_launch(ctx);
        if (s != MO_OK) return s;
    } else {
        // spatial ordering of this pass (performance only): cell keys, counting sort, tile bounding boxes
        enc_key_kernel<<<ctx->npsum, ON_BLOCK, 0, ctx->stream>>>(ctx->enc, ctx->nb, ctx->nbPad, ctx->npsum);
        s = post_launch(ctx);
        if (s != MO_OK) return s;
        enc_sortscatter_kernel<<<ctx->npsum, ON_BLOCK, 0, ctx->stream>>>(ctx->enc, ctx->nb, ctx->nbPad);
        s = post_launch(ctx);
        if (s != MO_OK) return s;
        enc_tilebox_kernel<<<ctx->nTiles, TJ, 0, ctx->stream>>>(ctx->enc, ctx->nbig);
        s = post_launch(ctx);
        if (s != MO_OK) return s;
        enc_find_kernel<<<dim3(ctx->nTiles, ctx->enc_split), CTA_THREADS, 0, ctx->stream>>>(fp);
        s = post_launch(ctx);
        if (s != MO_OK) return s;
    }
    // rows >= nbig hold no hits: only the tiles of the big rows are scanned
    enc_scan_kernel<<<ctx->nSrcTiles, TJ, 0, ctx->stream>>>(ctx->enc, ctx->nSrcTiles, ctx->cap, step_inc, ctx->dstats);
    s = post_launch(ctx);
    if (s != MO_OK) return s;
    const int pblocks = ctx->nsm * 2;
    enc_scatter_kernel<<<pblocks, 256, 0, ctx->stream>>>(ctx->enc, ctx->flag);
    s = post_launch(ctx);
    if (s != MO_OK) return s;
    enc_rank_kernel<<<pblocks, 256, 0, ctx->stream>>>(ctx->enc, ctx->pairs);
    s = post_launch(ctx);
    if (s != MO_OK) return s;
    EncWriteParams wp;
    wp.s = es; wp.e = ctx->enc; wp.pairs = ctx->pairs; wp.cap = ctx->cap; wp.flag = ctx->flag;
    int blocks = (ctx->nbig + 7) / 8;
    const int maxb = ctx->nsm;            // it exits at once unless count > cap: keep the empty launch small
    if (blocks > maxb) blocks = maxb;
    enc_write_kernel<<<blocks, 256, 0, ctx->stream>>>(wp);   // exits at once unless count > cap
    return post_launch(ctx);
}

// rcrit <- n_hill * r_H from the current x (and v for the osculating variant)
static mo_status enqueue_hill(mo_ctx* ctx, double n_hill, int mode, double* rhill) {
    double* rc = const_cast<double*>(ctx->rcrit);
    if (mode == 1) {   // heliocentric velocities need sum gm v
        kick_psum_kernel<false><<<ctx->npsum, ON_BLOCK, 0, ctx->stream>>>(ctx->v, nullptr, ctx->gm, ctx->nb, ctx->ld, 0.0, ctx->psumA, ctx->ticket);
        mo_status s = post_launch(ctx);
        if (s != MO_OK) return s;
        hill_kernel<1><<<ctx->npsum, ON_BLOCK, 0, ctx->stream>>>(ctx->x, ctx->v, ctx->gm, ctx->psumA, ctx->npsum, ctx->mu, n_hill, ctx->nb, ctx->ld, rc, rhill);
    } else {
        hill_kernel<0><<<ctx->npsum, ON_BLOCK, 0, ctx->stream>>>(ctx->x, ctx->v, ctx->gm, ctx->psumA, ctx->npsum, ctx->mu, n_hill, ctx->nb, ctx->ld, rc, rhill);
    }
    return post_launch(ctx);
}

// grids of the resolve kernels: class 0 (components of up to 63 pairs, 64 threads: several CTAs per SM), the larger
// classes hold few components (the stars around the big bodies): small grids, cheap to launch when they have nothing to do
static constexpr int RES_GRID_0_PER_SM = 6, RES_GRID_4 = 16, RES_GRID_S_PER_SM = 4;
static constexpr int RES_CL_GRID = RES_NCOL * (RES_NCLUSTERS / 3);   // classes 1..3: 8 clusters of 8 CTAs each

static mo_status ensure_resolve_scratch(mo_ctx* ctx) {
    if (ctx->res_loc) return MO_OK;
    const size_t capn = (size_t)(ctx->cap > 0 ? ctx->cap : 1);
    cudaError_t e = dalloc(ctx, &ctx->res_loc, (size_t)ctx->nb);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->res_out, 1);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->res_label, (size_t)ctx->nb);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->res_aux, (size_t)ctx->nb);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->fix_list, (size_t)ctx->nb);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->fix_nf, 1);
    if (e == cudaSuccess && ctx->use_sym) e = dalloc(ctx, &ctx->fix_part, (size_t)FIX_JS * 3 * ctx->nb);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->res_cown, capn);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->res_ckey, capn);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->res_cnp, capn);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->res_cstart, capn);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->res_cfill, capn);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->res_cq, capn);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->res_clist, capn * RES_NCLS);
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->res_ctl, (size_t)((RES_CTL_N + 15) & ~15));
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->res_tab, (size_t)6 * RES_KMAX * 1024 * RES_CL_GRID);   // per CTA of the widest launch
    if (e == cudaSuccess) e = dalloc(ctx, &ctx->res_mode, 2);
    if (e == cudaSuccess) { const int one[2] = {1, 1}; e = cudaMemcpyAsync(ctx->res_mode, one, sizeof(one), cudaMemcpyHostToDevice, ctx->stream); if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream); }
    // class D pools: every body and every pair of the list can be in a class-D component
    ctx->res_dbodyN = (long long)ctx->nb < 2 * (long long)capn ? (long long)ctx->nb : 2 * (long long)capn;
    if (ctx->cap > RES_PHI_3) {          // a shorter list cannot hold a class-D component
        if (e == cudaSuccess) e = dalloc(ctx, &ctx->res_dbody, (size_t)ctx->res_dbodyN * RES_D_BODY_PLANES);
        if (e == cudaSuccess) e = dalloc(ctx, &ctx->res_dbodyi, (size_t)ctx->res_dbodyN * RES_D_BODY_IPLANES);
        if (e == cudaSuccess) e = dalloc(ctx, &ctx->res_dpair, capn * RES_D_PAIR_PLANES);
        if (e == cudaSuccess) e = dalloc(ctx, &ctx->res_dpairi, capn * RES_D_PAIR_IPLANES);
    }
    // dynamic shared memory: 86 B per pair + 24 B per 32 pairs, 129 B per body, 6 * RES_KMAX doubles per body of tableau
    ctx->res_smemA = 88 * 64 + (132 + 6 * RES_KMAX * 8) * 64;
    ctx->res_smemB = 88 * 256 + (132 + 6 * RES_KMAX * 8) * 256;
    ctx->res_smemC = 227 * 1024 - 2048;                              // classes 2, 3: all there is (minus the static part)
    if (e == cudaSuccess) e = cudaFuncSetAttribute(resolve_solve_kernel<64, 0, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, ctx->res_smemA);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(resolve_solve_kernel<256, 1, RES_NCOL>, cudaFuncAttributeMaxDynamicSharedMemorySize, ctx->res_smemB);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(resolve_solve_kernel<512, 2, RES_NCOL>, cudaFuncAttributeMaxDynamicSharedMemorySize, ctx->res_smemC);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(resolve_solve_kernel<1024, 3, RES_NCOL>, cudaFuncAttributeMaxDynamicSharedMemorySize, ctx->res_smemC);
    if (e == cudaSuccess) e = cudaMemsetAsync(ctx->res_out, 0, sizeof(ResStats), ctx->stream);
    if (e == cudaSuccess) e = cudaMallocHost(reinterpret_cast<void**>(&ctx->res_host), sizeof(ResStats));
    for (int k = 0; k < 5 && e == cudaSuccess; ++k) {
        int plo = 0, phi = 0;
        cudaDeviceGetStreamPriorityRange(&plo, &phi);
        e = cudaStreamCreateWithPriority(&ctx->res_stream[k], cudaStreamNonBlocking, phi);   // ahead of a pair sum that becomes eligible at the same time
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->res_join[k], cudaEventDisableTiming);
    }
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->res_fork, cudaEventDisableTiming);
    if (e != cudaSuccess) { cudaGetLastError(); ctx->last_err = e; return e == cudaErrorMemoryAllocation ? MO_ENOMEM : MO_ECUDA; }
    return MO_OK;
}

static mo_status enqueue_resolve(mo_ctx* ctx, double dt, double tol) {
    StageRange nv("mopal: encounter resolution (f3)");
    ResParams rp;
    rp.x0 = ctx->x0; rp.v0 = ctx->v0; rp.x = ctx->x; rp.v = ctx->v; rp.gm = ctx->gm; rp.rcrit = ctx->rcrit;
    rp.pairs = ctx->pairs; rp.st = ctx->dstats; rp.out = ctx->res_out; rp.loc = ctx->res_loc; rp.label = ctx->res_label; rp.aux = ctx->res_aux; rp.cown = ctx->res_cown; rp.ckey = ctx->res_ckey;
    rp.cnp = ctx->res_cnp; rp.cstart = ctx->res_cstart; rp.cfill = ctx->res_cfill; rp.cq = ctx->res_cq; rp.clist = ctx->res_clist;
    rp.ctl = ctx->res_ctl; rp.mode = ctx->res_mode; rp.tab = ctx->res_tab; rp.dbody = ctx->res_dbody; rp.dbodyi = ctx->res_dbodyi; rp.dpair = ctx->res_dpair;
    rp.dpairi = ctx->res_dpairi; rp.dbodyN = ctx->res_dbodyN;
    rp.cap = ctx->cap > 0 ? ctx->cap : 1; rp.nb = ctx->nb; rp.ld = ctx->ld; rp.mu = ctx->mu; rp.h = dt; rp.tol = tol;
    {
        // one cluster of RES_LABEL_CTAS CTAs (a short list is handled by its first CTA alone)
        cudaLaunchConfig_t cfg = {};
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = RES_LABEL_CTAS; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.gridDim = dim3(RES_LABEL_CTAS); cfg.blockDim = dim3(RES_LABEL_THREADS); cfg.stream = ctx->stream; cfg.attrs = at; cfg.numAttrs = 1;
        CK(cudaLaunchKernelEx(&cfg, resolve_label_kernel, rp));
    }
    mo_status s = post_launch(ctx);
    if (s != MO_OK) return s;
    // the size classes side by side: the few large components (a giant's star is a long chain of right-hand sides on one
    // CTA) on streams of their own, the many small ones on the caller's
    cudaStream_t mainS = ctx->stream;
    CK(cudaEventRecord(ctx->res_fork, mainS));
    for (int k = 0; k < 5; ++k) {
        if (k == 0 && !ctx->res_dbody) continue;
        cudaStream_t st = ctx->res_stream[k];
        CK(cudaStreamWaitEvent(st, ctx->res_fork, 0));
        if (k == 0) resolve_stream_kernel<<<RES_GRID_4, RES_D_THREADS, 0, st>>>(rp);
        else if (k == 4) resolve_solve_kernel<64, 0, 1><<<ctx->nsm * RES_GRID_0_PER_SM, 64, ctx->res_smemA, st>>>(rp, ctx->res_smemA);
        else {
            // clusters of RES_NCOL CTAs: one component per cluster, one Bulirsch-Stoer column per CTA
            cudaLaunchConfig_t cfg = {};
            cudaLaunchAttribute at[1];
            at[0].id = cudaLaunchAttributeClusterDimension;
            at[0].val.clusterDim.x = RES_NCOL; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
            cfg.gridDim = dim3(RES_CL_GRID); cfg.stream = st; cfg.attrs = at; cfg.numAttrs = 1;
            if (k == 1) { cfg.blockDim = dim3(1024); cfg.dynamicSmemBytes = ctx->res_smemC; CK(cudaLaunchKernelEx(&cfg, resolve_solve_kernel<1024, 3, RES_NCOL>, rp, ctx->res_smemC)); }
            else if (k == 2) { cfg.blockDim = dim3(512); cfg.dynamicSmemBytes = ctx->res_smemC; CK(cudaLaunchKernelEx(&cfg, resolve_solve_kernel<512, 2, RES_NCOL>, rp, ctx->res_smemC)); }
            else { cfg.blockDim = dim3(256); cfg.dynamicSmemBytes = ctx->res_smemB; CK(cudaLaunchKernelEx(&cfg, resolve_solve_kernel<256, 1, RES_NCOL>, rp, ctx->res_smemB)); }
        }
        s = post_launch(ctx);
        if (s != MO_OK) return s;
        CK(cudaEventRecord(ctx->res_join[k], st));
    }
    // the small systems (almost all of them) on the caller's stream: one CTA of 8 warps each, a column per warp
    resolve_small_kernel<<<ctx->nsm * RES_GRID_S_PER_SM, RES_S_THREADS, 0, mainS>>>(rp);
    s = post_launch(ctx);
    if (s != MO_OK) return s;
    for (int k = 0; k < 5; ++k) {
        if (k == 0 && !ctx->res_dbody) continue;
        CK(cudaStreamWaitEvent(mainS, ctx->res_join[k], 0));
    }
    return MO_OK;
}

static mo_status enqueue_step(mo_ctx* ctx, double dt) {
    StageRange nv("mopal: hybrid step (a9)");
    if (ctx->use_small && ctx->res_tol <= 0.0) {
        SmallParams q;
        MidParams& mp = q.m;
        mp.x = ctx->x; mp.v = ctx->v; mp.x0 = ctx->x0; mp.v0 = ctx->v0; mp.gm = ctx->gm; mp.rcrit = ctx->rcrit;
        mp.x1 = nullptr; mp.v1 = nullptr;
        mp.psum_in = nullptr; mp.psum_out = nullptr; mp.ticket = nullptr; mp.enc = ctx->enc; mp.flag = ctx->flag;
        mp.st = ctx->dstats; mp.nb = ctx->nb; mp.ld = ctx->ld; mp.nbPad = ctx->nbPad; mp.npsum = 0; mp.nbig = ctx->nbig;
        mp.hj_over_mu = 0.5 * dt / ctx->mu; mp.mu = ctx->mu; mp.h = dt;
        q.a = ctx->a; q.hk = 0.5 * dt; q.pairs = ctx->pairs; q.cap = ctx->cap;
        q.hill_mode = ctx->hill_mode; q.hill_n = ctx->hill_n;
        int thr = (ctx->nb + 31) / 32 * 32;
        if (thr < 64) thr = 64;
        step_small_kernel<<<1, thr, 0, ctx->stream>>>(q);
        mo_status ss = post_launch(ctx);
        if (ss != MO_OK) return ss;
        return enqueue_accel(ctx, false, 0.0, true, 0.5 * dt);   // both jumps are done: a(x), closing kick
    }
    if (ctx->hill_mode >= 0) {
        mo_status hs = enqueue_hill(ctx, ctx->hill_n, ctx->hill_mode, nullptr);
        if (hs != MO_OK) return hs;
    }
    nvtxRangePushA("mopal: kick, sum gm v, jump, snapshot, drift, boxes (a3-a7)");
    kick_psum_kernel<true><<<ctx->npsum, ON_BLOCK, 0, ctx->stream>>>(ctx->v, ctx->a, ctx->gm, ctx->nb, ctx->ld, 0.5 * dt, ctx->psumA, ctx->ticket);
    mo_status s = post_launch(ctx);
    if (s != MO_OK) { nvtxRangePop(); return s; }
    MidParams mp;
    mp.x = ctx->x; mp.v = ctx->v; mp.x0 = ctx->x0; mp.v0 = ctx->v0; mp.gm = ctx->gm; mp.rcrit = ctx->rcrit;
    mp.psum_in = ctx->psumA; mp.psum_out = ctx->psumB; mp.ticket = ctx->ticket + 1;
    // with the encounter solve: beside the pair sum when the two-sided kernel runs (fixup.cuh), else before it
    const bool ovl_res = ctx->overlap && ctx->res_tol > 0.0 && ctx->use_sym && ctx->shard_world == 1 && ctx->fix_part;
    const bool ovl = (ctx->overlap && ctx->res_tol <= 0.0) || ovl_res;
    mp.x1 = ovl ? ctx->x1 : nullptr; mp.v1 = ovl ? ctx->v1 : nullptr; mp.enc = ctx->enc; mp.flag = ctx->flag;
    mp.st = ctx->dstats; mp.nb = ctx->nb; mp.ld = ctx->ld; mp.nbPad = ctx->nbPad; mp.npsum = ctx->npsum;
    mp.nbig = ctx->nbig;
    mp.hj_over_mu = 0.5 * dt / ctx->mu; mp.mu = ctx->mu; mp.h = dt;
    jump_drift_boxes_kernel<<<ctx->npsum, ON_BLOCK, 0, ctx->stream>>>(mp);
    s = post_launch(ctx);
    nvtxRangePop();
    if (s != MO_OK) return s;
    if (ovl_res) {
        // fork: encounter pass + encounter solve on enc_stream (read x0, v0, x1, v1; the solve writes x, v of the flagged
        // bodies), pair sum over the drifted positions x1 on the main stream; join; corrections, jump, kick
        cudaStream_t mainS = ctx->stream;
        mode_latch_kernel<<<1, 1, 0, mainS>>>(ctx->res_mode);
        s = post_launch(ctx);
        if (s != MO_OK) return s;
        CK(cudaEventRecord(ctx->ev_fork, mainS));
        CK(cudaStreamWaitEvent(ctx->enc_stream, ctx->ev_fork, 0));
        EncState es = enc_state(ctx, ctx->x0, ctx->v0, dt);
        es.x1 = ctx->x1; es.v1 = ctx->v1;
        ctx->stream = ctx->enc_stream;
        s = enqueue_pairs(ctx, es, 1);
        if (s == MO_OK) {       // the list of the flagged bodies for the corrections below: the flags are final here
            fix_list_kernel<<<1, FIX_LIST_THREADS, 0, ctx->stream>>>(ctx->flag, ctx->nb, ctx->fix_list, ctx->fix_nf, Gate{ctx->res_mode, 1});
            s = post_launch(ctx);
        }
        if (s == MO_OK) s = enqueue_resolve(ctx, dt, ctx->res_tol);
        ctx->stream = mainS;
        if (s != MO_OK) return s;
        CK(cudaEventRecord(ctx->ev_join, ctx->enc_stream));
        // The pair sum in two launches.  A giant's star needs a whole SM for its CTA; inside one launch of 15 waves the pair
        // kernel's CTAs would keep every SM half full and the solve would wait for the tail.  So: the first tenth of the
        // units while the encounter pass and the label kernel run; the rest once the components are known (res_fork) - then
        // the solve's CTAs and the pair kernel's become eligible together on draining SMs, and the solve's streams have the
        // higher priority.
        const Gate gO = {ctx->res_mode, 1}, gS = {ctx->res_mode, 0};   // beside the pair sum / before it (see below)
        ctx->pair_x = ctx->x1; ctx->gate = gO;
        pack_kernel<false, true><<<ctx->nSrcTiles, TJ, 0, mainS>>>(ctx->x1, ctx->gm, ctx->rcrit, ctx->nb, ctx->nbig, ctx->ld, ctx->tiles, nullptr, 0, 0.0, gO);
        s = post_launch(ctx);
        // (a tenth of the WORK: the units differ in length)
        const int ucut = (int)(std::lower_bound(ctx->h_uwork.begin(), ctx->h_uwork.end() - 1, ctx->h_uwork.back() / 10) - ctx->h_uwork.begin());
        if (s == MO_OK) { ctx->pair_u0 = 0; ctx->pair_u1 = ucut; s = launch_pair(ctx); }
        if (s == MO_OK) {
            CK(cudaStreamWaitEvent(mainS, ctx->res_fork, 0));
            ctx->pair_u0 = ucut; ctx->pair_u1 = ctx->sym_nunits; s = launch_pair(ctx);
        }
        ctx->pair_x = nullptr; ctx->pair_u0 = ctx->pair_u1 = -1; ctx->gate = Gate{nullptr, 0};
        if (s != MO_OK) return s;
        sym_reduce_kernel<false, false><<<dim3((ctx->nb + 31) / 32, 3), RED_THREADS, 0, mainS>>>(ctx->sym_partI, ctx->sym_partJ, ctx->sym_ustart, ctx->nb, ctx->ld, ctx->nbPad,
                                                                                ctx->a, nullptr, 0.0, 0, ctx->sym_nunits, nullptr, sym_rows(ctx->sym_ipt), gO);
        s = post_launch(ctx);
        if (s != MO_OK) return s;
        CK(cudaStreamWaitEvent(mainS, ctx->ev_join, 0));
        kick_psum_kernel<false><<<ctx->npsum, ON_BLOCK, 0, mainS>>>(ctx->v, nullptr, ctx->gm, ctx->nb, ctx->ld, 0.0, ctx->psumB, ctx->ticket + 1);
        s = post_launch(ctx);
        if (s != MO_OK) return s;
        FixParams fp;
        fp.x = ctx->x; fp.x1 = ctx->x1; fp.gm = ctx->gm; fp.rcrit = ctx->rcrit; fp.flag = ctx->flag; fp.flist = ctx->fix_list; fp.nf = ctx->fix_nf;
        fp.a = ctx->a; fp.part = ctx->fix_part; fp.nb = ctx->nb; fp.ld = ctx->ld; fp.gate = gO;
        fix_unflagged_kernel<<<(ctx->nb + FIX_UT / FIX_SP - 1) / (FIX_UT / FIX_SP), FIX_UT, 0, mainS>>>(fp);
        s = post_launch(ctx);
        if (s != MO_OK) return s;
        // (the number of flagged bodies is not known on the host: CTAs beyond the list exit at once)
        const int fgx = (ctx->nb + FIX_FB - 1) / FIX_FB < 512 ? (ctx->nb + FIX_FB - 1) / FIX_FB : 512;
        fix_flagged_kernel<<<dim3(fgx, FIX_JS), FIX_THREADS, 0, mainS>>>(fp);
        s = post_launch(ctx);
        if (s != MO_OK) return s;
        fix_flagged_reduce_kernel<<<(ctx->nb + FIX_THREADS - 1) / FIX_THREADS, FIX_THREADS, 0, mainS>>>(fp);
        s = post_launch(ctx);
        if (s != MO_OK) return s;
        jump_kick_kernel<<<ctx->npsum, ON_BLOCK, 0, mainS>>>(ctx->x, ctx->v, ctx->a, ctx->psumB, ctx->npsum, 0.5 * dt / ctx->mu, 0.5 * dt, ctx->nb, ctx->ld, gO);
        s = post_launch(ctx);
        if (s != MO_OK) return s;
        // the other way, for lists without a long chain (only components of up to 63 pairs: their solve takes tens of
        // microseconds, less than the exchange of the flagged bodies' terms costs): jump, pair sum over the resolved
        // positions, kick.  Both ways are in the graph; which one works is the device flag the label kernel of the LAST
        // step set (latched at the start of this step) - a stale choice costs time, never correctness.
        ctx->gate = gS;
        s = enqueue_accel(ctx, true, 0.5 * dt, true, 0.5 * dt);
        ctx->gate = Gate{nullptr, 0};
        return s;
    }
    if (ovl) {
        // fork: encounter pass on enc_stream (reads x0, v0, x1, v1, boxes, rcrit; writes pairs, flag, stats),
        // jump + pair sum + closing kick on the main stream (moves x, v; writes a); join at the end
        cudaStream_t mainS = ctx->stream;
        CK(cudaEventRecord(ctx->ev_fork, mainS));
        CK(cudaStreamWaitEvent(ctx->enc_stream, ctx->ev_fork, 0));
        EncState es = enc_state(ctx, ctx->x0, ctx->v0, dt);
        es.x1 = ctx->x1; es.v1 = ctx->v1;
        ctx->stream = ctx->enc_stream;
        s = enqueue_pairs(ctx, es, 1);
        ctx->stream = mainS;
        if (s != MO_OK) return s;
        CK(cudaEventRecord(ctx->ev_join, ctx->enc_stream));
        s = enqueue_accel(ctx, true, 0.5 * dt, true, 0.5 * dt);
        if (s != MO_OK) return s;
        CK(cudaStreamWaitEvent(mainS, ctx->ev_join, 0));
        return MO_OK;
    }
    s = enqueue_pairs(ctx, enc_state(ctx, ctx->x0, ctx->v0, dt), 1);
    if (s != MO_OK) return s;
    if (ctx->res_tol > 0.0) {
        s = enqueue_resolve(ctx, dt, ctx->res_tol);
        if (s != MO_OK) return s;
        // v of the resolved bodies changed: sum gm v for the second jump again
        kick_psum_kernel<false><<<ctx->npsum, ON_BLOCK, 0, ctx->stream>>>(ctx->v, nullptr, ctx->gm, ctx->nb, ctx->ld, 0.0, ctx->psumB, ctx->ticket + 1);
        s = post_launch(ctx);
        if (s != MO_OK) return s;
    }
    return enqueue_accel(ctx, true, 0.5 * dt, true, 0.5 * dt);
}

static mo_status read_stats(mo_ctx* ctx, mo_stats* out, bool* overflow) {
    CK(cudaMemcpyAsync(ctx->hstats, ctx->dstats, sizeof(DevStats), cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    if (out) {
        out->steps_done = ctx->hstats->steps_done;
        out->nce_last = ctx->hstats->nce_last;
        out->nce_total = ctx->hstats->nce_total;
        out->drift_fail = ctx->hstats->drift_fail;
        out->max_newton = ctx->hstats->max_newton;
        out->resolve_fail = ctx->hstats->resolve_fail;
        out->reserved = 0;
    }
    if (overflow) *overflow = ctx->hstats->overflow != 0;
    return MO_OK;
}

static mo_status status_from_stats(mo_ctx* ctx, mo_stats* out) {
    bool ovf = false;
    mo_stats tmp;
    mo_status s = read_stats(ctx, &tmp, &ovf);
    if (s != MO_OK) return s;
    if (out) *out = tmp;
    if (ovf) return MO_EOVERFLOW;
    if (tmp.drift_fail > 0) return MO_ENOCONV;
    if (tmp.resolve_fail > 0) return MO_ERESOLVE;
    return MO_OK;
}

// ---- public entry points ---------------------------------------------------------------------
extern "C" mo_status mo_accel(mo_ctx* ctx) {
    if (!ctx) return MO_EINVAL;
    mo_status s = ensure_pair_scratch(ctx);
    if (s != MO_OK) return s;
    s = enqueue_accel(ctx, false, 0.0, false, 0.0);
    if (s == MO_OK) ctx->a_valid = ctx->shard_world == 1;     // sharded: a share, until mo_accel_summed
    return s;
}

extern "C" mo_status mo_drift(mo_ctx* ctx, double dt) {
    if (!ctx || !isfinite(dt)) return MO_EINVAL;
    const int nblk = (ctx->nb + ON_BLOCK - 1) / ON_BLOCK;
    drift_kernel<<<nblk, ON_BLOCK, 0, ctx->stream>>>(ctx->x, ctx->v, ctx->nb, ctx->ld, ctx->mu, dt, ctx->dstats);
    ctx->a_valid = false;
    return post_launch(ctx);
}

extern "C" mo_status mo_snapshot(mo_ctx* ctx) {
    if (!ctx) return MO_EINVAL;
    const size_t bytes = 3 * (size_t)ctx->ld * sizeof(double);
    CK(cudaMemcpyAsync(ctx->x0, ctx->x, bytes, cudaMemcpyDeviceToDevice, ctx->stream));
    CK(cudaMemcpyAsync(ctx->v0, ctx->v, bytes, cudaMemcpyDeviceToDevice, ctx->stream));
    ctx->snap_valid = true;
    return MO_OK;
}

extern "C" mo_status mo_snapshot_ptrs(mo_ctx* ctx, const double** x0, const double** v0) {
    if (!ctx) return MO_EINVAL;
    if (x0) *x0 = ctx->x0;
    if (v0) *v0 = ctx->v0;
    return MO_OK;
}

extern "C" mo_status mo_snapshot_copy(mo_ctx* ctx, double* x0_dst, double* v0_dst) {
    if (!ctx || !x0_dst || !v0_dst) return MO_EINVAL;
    const size_t bytes = 3 * (size_t)ctx->ld * sizeof(double);
    CK(cudaMemcpyAsync(x0_dst, ctx->x0, bytes, cudaMemcpyDeviceToDevice, ctx->stream));
    CK(cudaMemcpyAsync(v0_dst, ctx->v0, bytes, cudaMemcpyDeviceToDevice, ctx->stream));
    return MO_OK;
}

extern "C" mo_status mo_boxes_copy(mo_ctx* ctx, double* box_dst) {
    if (!ctx || !box_dst || !ctx->box_valid) return MO_EINVAL;
    CK(cudaMemcpyAsync(box_dst, ctx->enc.box, (size_t)ctx->nb * sizeof(double4), cudaMemcpyDeviceToDevice, ctx->stream));
    return MO_OK;
}

extern "C" mo_status mo_set_nbig(mo_ctx* ctx, int32_t nbig) {
    if (!ctx || nbig < 1 || nbig > ctx->nb) return MO_EINVAL;
    if (nbig == ctx->nbig) return MO_OK;
    CK(cudaStreamSynchronize(ctx->stream));   // nothing in flight may still use the scratch freed below
    if (ctx->gexec) { cudaGraphExecDestroy(ctx->gexec); ctx->gexec = nullptr; }
    cudaFree(ctx->part); ctx->part = nullptr;
    cudaFree(ctx->sym_units); cudaFree(ctx->sym_ustart); cudaFree(ctx->sym_partI); cudaFree(ctx->sym_partJ); cudaFree(ctx->sym_qr);
    ctx->sym_qr = nullptr;
    ctx->sym_units = nullptr; ctx->sym_ustart = nullptr; ctx->sym_partI = nullptr; ctx->sym_partJ = nullptr;
    ctx->pair_ready = false;
    ctx->a_valid = false;
    ctx->nbig = nbig;
    ctx->nSrcTiles = (nbig + TJ - 1) / TJ;
    choose_geometry(ctx);
    if (ctx->shard_world > 1 && !(ctx->use_sym || ctx->use_big)) {     // this size takes a kernel that does not split its work
        ctx->shard_rank = 0; ctx->shard_world = 1;
        return MO_EINVAL;
    }
    return MO_OK;
}

extern "C" mo_status mo_resolve(mo_ctx* ctx, double dt, double tol) {
    if (!ctx || !isfinite(dt) || dt == 0.0 || !(tol > 0.0) || !ctx->snap_valid) return MO_EINVAL;
    mo_status s = ensure_resolve_scratch(ctx);
    if (s != MO_OK) return s;
    return enqueue_resolve(ctx, dt, tol);
}

extern "C" mo_status mo_set_resolve(mo_ctx* ctx, double tol) {
    if (!ctx || !isfinite(tol)) return MO_EINVAL;
    if (tol > 0.0) {
        mo_status s = ensure_resolve_scratch(ctx);
        if (s != MO_OK) return s;
    }
    if (ctx->gexec) {
        CK(cudaStreamSynchronize(ctx->stream));
        cudaGraphExecDestroy(ctx->gexec); ctx->gexec = nullptr;
    }
    ctx->res_tol = tol > 0.0 ? tol : 0.0;
    return MO_OK;
}

extern "C" mo_status mo_resolve_stats(mo_ctx* ctx, int32_t* out4) {
    if (!ctx || !out4) return MO_EINVAL;
    if (!ctx->res_out) { out4[0] = out4[1] = out4[2] = out4[3] = 0; return MO_OK; }
    CK(cudaMemcpyAsync(ctx->res_host, ctx->res_out, sizeof(ResStats), cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    out4[0] = ctx->res_host->bodies; out4[1] = ctx->res_host->steps; out4[2] = ctx->res_host->rhs; out4[3] = ctx->res_host->fail;
    return MO_OK;
}

extern "C" mo_status mo_hill(mo_ctx* ctx, double n_hill, int32_t mode, double* rhill_dev) {
    if (!ctx || !isfinite(n_hill) || n_hill < 0.0 || (mode != 0 && mode != 1)) return MO_EINVAL;
    ctx->a_valid = false;             // K depends on rcrit
    return enqueue_hill(ctx, n_hill, mode, rhill_dev);
}

extern "C" mo_status mo_set_hill(mo_ctx* ctx, double n_hill, int32_t mode) {
    if (!ctx || mode < -1 || mode > 1 || (mode >= 0 && (!isfinite(n_hill) || n_hill < 0.0))) return MO_EINVAL;
    if (ctx->gexec) {
        CK(cudaStreamSynchronize(ctx->stream));
        cudaGraphExecDestroy(ctx->gexec); ctx->gexec = nullptr;
    }
    ctx->hill_mode = mode;
    if (mode >= 0) ctx->hill_n = n_hill;
    return MO_OK;
}

static mo_status vshift(mo_ctx* ctx, bool to_dh) {
    kick_psum_kernel<false><<<ctx->npsum, ON_BLOCK, 0, ctx->stream>>>(ctx->v, nullptr, ctx->gm, ctx->nb, ctx->ld, 0.0, ctx->psumA, ctx->ticket);
    mo_status s = post_launch(ctx);
    if (s != MO_OK) return s;
    if (to_dh)
        vshift_kernel<true><<<ctx->npsum, ON_BLOCK, 0, ctx->stream>>>(ctx->v, ctx->psumA, ctx->npsum, ctx->gmsum, ctx->mu, ctx->nb, ctx->ld);
    else
        vshift_kernel<false><<<ctx->npsum, ON_BLOCK, 0, ctx->stream>>>(ctx->v, ctx->psumA, ctx->npsum, ctx->gmsum, ctx->mu, ctx->nb, ctx->ld);
    return post_launch(ctx);
}
extern "C" mo_status mo_h2dh(mo_ctx* ctx) { return ctx ? vshift(ctx, true) : MO_EINVAL; }
extern "C" mo_status mo_dh2h(mo_ctx* ctx) { return ctx ? vshift(ctx, false) : MO_EINVAL; }

extern "C" mo_status mo_energy(mo_ctx* ctx, mo_energy_t* out_host) {
    if (!ctx || !out_host) return MO_EINVAL;
    const int nIb = (ctx->nbig + EN_T - 1) / EN_T;
    const int nT = (ctx->nb + EN_T - 1) / EN_T;
    int split = (32 * ctx->nsm + nIb - 1) / nIb;         // many short CTAs: the rows of the triangle differ in length
    if (split > nT) split = nT;
    if (split < 1) split = 1;
    if (!ctx->en_on || ctx->en_npair != nIb * split) {   // (re)allocate after mo_set_nbig
        cudaFree(ctx->en_pair); ctx->en_pair = nullptr;
        cudaError_t e = cudaSuccess;
        if (!ctx->en_on) e = dalloc(ctx, &ctx->en_on, (size_t)ctx->npsum * EN_NSUM);
        if (e == cudaSuccess && !ctx->en_out) e = dalloc(ctx, &ctx->en_out, 8);
        if (e == cudaSuccess && !ctx->en_host) e = cudaMallocHost(reinterpret_cast<void**>(&ctx->en_host), 8 * sizeof(double));
        if (e == cudaSuccess) e = dalloc(ctx, &ctx->en_pair, (size_t)nIb * split);
        if (e != cudaSuccess) { cudaGetLastError(); ctx->last_err = e; return e == cudaErrorMemoryAllocation ? MO_ENOMEM : MO_ECUDA; }
        ctx->en_npair = nIb * split; ctx->en_split = split;
    }
    energy_on_kernel<<<ctx->npsum, ON_BLOCK, 0, ctx->stream>>>(ctx->x, ctx->v, ctx->gm, ctx->nb, ctx->ld, ctx->en_on);
    mo_status s = post_launch(ctx);
    if (s != MO_OK) return s;
    energy_pair_kernel<<<dim3(nIb, split), EN_T, 0, ctx->stream>>>(ctx->x, ctx->gm, ctx->nb, ctx->nbig, ctx->ld, ctx->en_pair);
    s = post_launch(ctx);
    if (s != MO_OK) return s;
    energy_final_kernel<<<1, 256, 0, ctx->stream>>>(ctx->en_on, ctx->npsum, ctx->en_pair, ctx->en_npair, ctx->mu, ctx->en_out);
    s = post_launch(ctx);
    if (s != MO_OK) return s;
    CK(cudaMemcpyAsync(ctx->en_host, ctx->en_out, 7 * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    const double G = ctx->G;
    out_host->T = ctx->en_host[0] / G; out_host->Us = ctx->en_host[1] / G; out_host->Up = ctx->en_host[2] / G;
    out_host->E = ctx->en_host[3] / G;
    for (int c = 0; c < 3; ++c) out_host->L[c] = ctx->en_host[4 + c] / G;
    return MO_OK;
}

extern "C" mo_status mo_invalidate_accel(mo_ctx* ctx) {
    if (!ctx) return MO_EINVAL;
    ctx->a_valid = false;
    return MO_OK;
}

extern "C" mo_status mo_encounters(mo_ctx* ctx, double dt, const double* x0, const double* v0, int64_t* count_host) {
    if (!ctx || !isfinite(dt) || dt == 0.0) return MO_EINVAL;
    if ((x0 == nullptr) != (v0 == nullptr)) return MO_EINVAL;
    if (!x0) {
        if (!ctx->snap_valid) return MO_EINVAL;
        x0 = ctx->x0; v0 = ctx->v0;
    } else if (!aligned16(x0) || !aligned16(v0)) {
        return MO_EINVAL;
    }
    EncState es = enc_state(ctx, x0, v0, dt);
    boxes_kernel<<<(ctx->nbPad + ON_BLOCK - 1) / ON_BLOCK, ON_BLOCK, 0, ctx->stream>>>(es, ctx->enc, ctx->nbPad, ctx->flag);
    mo_status s = post_launch(ctx);
    if (s != MO_OK) return s;
    s = enqueue_pairs(ctx, es, 0);
    if (s != MO_OK) return s;
    ctx->box_valid = true;
    if (count_host) {
        mo_stats st;
        s = read_stats(ctx, &st, nullptr);
        if (s != MO_OK) return s;
        *count_host = st.nce_last;
        if (st.nce_last > ctx->cap) return MO_EOVERFLOW;
    }
    return MO_OK;
}

extern "C" mo_status mo_shard_range(int64_t n, int32_t rank, int32_t world, int64_t* lo, int64_t* hi) {
    if (n < 0 || world < 1 || rank < 0 || rank >= world || !lo || !hi) return MO_EINVAL;
    long long a, b;
    shard_range(n, rank, world, &a, &b);
    *lo = a; *hi = b;
    return MO_OK;
}

extern "C" mo_status mo_set_shard(mo_ctx* ctx, int32_t rank, int32_t world) {
    if (!ctx || world < 1 || rank < 0 || rank >= world) return MO_EINVAL;
    // only the kernels of the large systems split their work: the two-sided pair sum (nb > 2560) and the big x all sum
    if (world > 1 && !(ctx->use_sym || ctx->use_big)) return MO_EINVAL;
    if (ctx->gexec) {
        CK(cudaStreamSynchronize(ctx->stream));
        cudaGraphExecDestroy(ctx->gexec); ctx->gexec = nullptr;
    }
    ctx->shard_rank = rank; ctx->shard_world = world;
    ctx->a_valid = false;
    if (ctx->use_sym && ctx->pair_ready) CK(sym_fill_qr(ctx));
    return MO_OK;
}

extern "C" mo_status mo_shard_units(const mo_ctx* ctx, int64_t* units, int64_t* lo, int64_t* hi) {
    if (!ctx || !units || !lo || !hi) return MO_EINVAL;
    const long long n = ctx->use_sym ? ctx->sym_nunits : ctx->use_big ? ctx->nIblk : 0;
    long long a = 0, b = n;
    if (ctx->use_sym) sym_shard_units(ctx, &a, &b);
    else if (ctx->shard_world > 1) shard_range(n, ctx->shard_rank, ctx->shard_world, &a, &b);
    *units = n; *lo = a; *hi = b;
    return MO_OK;
}

// Sharded step, first part: everything up to and including this rank's share of the pair sum; a holds the share.
extern "C" mo_status mo_step_begin(mo_ctx* ctx, double dt) {
    if (!ctx || !isfinite(dt) || dt == 0.0 || ctx->shard_world < 2) return MO_EINVAL;
    if (!ctx->a_valid) return MO_EINVAL;          // mo_accel + the caller's sum over the ranks + mo_accel_summed come first
    mo_status s = ensure_pair_scratch(ctx);
    if (s != MO_OK) return s;
    s = enqueue_step(ctx, dt);
    if (s == MO_OK) { ctx->snap_valid = true; ctx->box_valid = true; ctx->a_valid = false; }
    return s;
}

// The caller has summed a over the ranks: a is the acceleration of the current x.
extern "C" mo_status mo_accel_summed(mo_ctx* ctx) {
    if (!ctx || ctx->shard_world < 2) return MO_EINVAL;
    ctx->a_valid = true;
    return MO_OK;
}

// Sharded step, second part (after the sum of a over the ranks): the closing kick.
extern "C" mo_status mo_step_end(mo_ctx* ctx, double dt, mo_stats* stats_host) {
    if (!ctx || !isfinite(dt) || dt == 0.0 || ctx->shard_world < 2) return MO_EINVAL;
    kick_psum_kernel<true><<<ctx->npsum, ON_BLOCK, 0, ctx->stream>>>(ctx->v, ctx->a, ctx->gm, ctx->nb, ctx->ld, 0.5 * dt, ctx->psumA, ctx->ticket);
    mo_status s = post_launch(ctx);
    if (s != MO_OK) return s;
    ctx->a_valid = true;
    if (stats_host) return status_from_stats(ctx, stats_host);
    return MO_OK;
}

extern "C" mo_status mo_step(mo_ctx* ctx, double dt, int32_t nsteps, mo_stats* stats_host) {
    if (!ctx || !isfinite(dt) || dt == 0.0 || nsteps < 0) return MO_EINVAL;
    if (ctx->shard_world > 1) return MO_EINVAL;   // sharded: mo_step_begin / sum of a over the ranks / mo_step_end
    mo_status s = ensure_pair_scratch(ctx);   // before any capture: allocation cannot be recorded
    if (s != MO_OK) return s;
    if (!ctx->a_valid && nsteps > 0) {
        s = mo_accel(ctx);
        if (s != MO_OK) return s;
    }
    const bool graph = ctx->use_graph && !ctx->timing && !ctx->debug && nsteps > 1;
    if (graph) {
        if (!ctx->gexec || ctx->gdt != dt) {
            if (ctx->gexec) { cudaGraphExecDestroy(ctx->gexec); ctx->gexec = nullptr; }
            cudaGraph_t g = nullptr;
            const long long l0 = ctx->launches;
            // the caller's stream may be the legacy default stream, which cannot be captured:
            // record the step on an owned stream, replay the graph on the caller's
            if (!ctx->cap_stream) CK(cudaStreamCreateWithFlags(&ctx->cap_stream, cudaStreamNonBlocking));
            cudaStream_t user = ctx->stream;
            CK(cudaStreamBeginCapture(ctx->cap_stream, cudaStreamCaptureModeThreadLocal));
            ctx->stream = ctx->cap_stream;
            s = enqueue_step(ctx, dt);
            ctx->stream = user;
            cudaError_t e = cudaStreamEndCapture(ctx->cap_stream, &g);
            ctx->gkernels = (int)(ctx->launches - l0);
            ctx->launches = l0;  // captured, not launched
            if (s != MO_OK || e != cudaSuccess) {
                if (g) cudaGraphDestroy(g);
                ctx->last_err = e;
                cudaGetLastError();
                return MO_ECUDA;
            }
            e = set_node_priorities(ctx, g);
            if (e == cudaSuccess) e = cudaGraphInstantiateWithFlags(&ctx->gexec, g, cudaGraphInstantiateFlagUseNodePriority);
            cudaGraphDestroy(g);
            if (e != cudaSuccess) { ctx->gexec = nullptr; ctx->last_err = e; return MO_ECUDA; }
            ctx->gdt = dt;
        }
        for (int k = 0; k < nsteps; ++k) {
            CK(cudaGraphLaunch(ctx->gexec, ctx->stream));
            ctx->launches += ctx->gkernels;
        }
    } else {
        for (int k = 0; k < nsteps; ++k) {
            s = enqueue_step(ctx, dt);
            if (s != MO_OK) return s;
        }
    }
    if (nsteps > 0) { ctx->snap_valid = true; ctx->a_valid = true; ctx->box_valid = true; }
    if (stats_host) return status_from_stats(ctx, stats_host);
    return MO_OK;
}

extern "C" mo_status mo_get_stats(mo_ctx* ctx, mo_stats* stats_host) {
    if (!ctx || !stats_host) return MO_EINVAL;
    return status_from_stats(ctx, stats_host);
}

extern "C" int64_t mo_launch_count(const mo_ctx* ctx) { return ctx ? ctx->launches : 0; }
extern "C" int64_t mo_workspace_bytes(const mo_ctx* ctx) { return ctx ? (int64_t)ctx->ws_bytes : 0; }

extern "C" mo_status mo_pair_geometry(const mo_ctx* ctx, int32_t* ipt, int32_t* jsplit, int32_t* ctas, int32_t* ctas_per_sm) {
    if (!ctx) return MO_EINVAL;
    if (ipt) *ipt = ctx->ipt;
    if (jsplit) *jsplit = ctx->nsplit;
    if (ctas) *ctas = ctx->use_sym ? ctx->sym_nunits : ctx->use_big ? ctx->big_grid : ctx->nIblk * ctx->nsplit;
    if (ctx->use_psm) {
        const int per = PSM_THREADS / ctx->psm_g;
        if (ipt) *ipt = 1;
        if (jsplit) *jsplit = ctx->psm_g;
        if (ctas) *ctas = (ctx->nb + per - 1) / per;
        if (ctas_per_sm) *ctas_per_sm = 4;
        return MO_OK;
    }
    if (ctx->use_sym && jsplit) *jsplit = ctx->sym_ch;
    if (ctas_per_sm) *ctas_per_sm = ctx->ctas_per_sm;
    return MO_OK;
}

extern "C" const char* mo_pair_kernel_name(const mo_ctx* ctx) {
    if (!ctx) return nullptr;
    return ctx->use_psm ? "pair_small_kernel" : ctx->use_big ? "pair_big_kernel" : ctx->use_sym ? "pair_sym_kernel" : "pair_accel_kernel";
}

extern "C" mo_status mo_set_kernel_timing(mo_ctx* ctx, int32_t on) {
    if (!ctx) return MO_EINVAL;
    ctx->timing = on != 0;
    ctx->ev_used = 0;
    return MO_OK;
}

extern "C" mo_status mo_pair_kernel_ms(mo_ctx* ctx, double* ms_out, int32_t* n_out) {
    if (!ctx || !ms_out) return MO_EINVAL;
    CK(cudaStreamSynchronize(ctx->stream));
    double tot = 0.0;
    int n = 0;
    for (size_t k = 0; k + 1 < ctx->ev_used; k += 2) {
        float ms = 0.f;
        CK(cudaEventElapsedTime(&ms, ctx->ev[k], ctx->ev[k + 1]));
        tot += ms; ++n;
    }
    *ms_out = n ? tot / n : 0.0;
    if (n_out) *n_out = n;
    ctx->ev_used = 0;
    return MO_OK;
}

extern "C" mo_status mo_step_host(mo_ctx* ctx, double dt, int32_t nsteps, double* x_host, double* v_host,
                                  const double* rcrit_host, int32_t a_is_current, int32_t* pairs_host, int64_t cap_host,
                                  mo_stats* stats_host) {
    if (!ctx || !x_host || !v_host || !isfinite(dt) || dt == 0.0 || nsteps < 0 || cap_host < 0) return MO_EINVAL;
    const size_t bytes = 3 * (size_t)ctx->ld * sizeof(double);
    CK(cudaMemcpyAsync(ctx->x, x_host, bytes, cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaMemcpyAsync(ctx->v, v_host, bytes, cudaMemcpyHostToDevice, ctx->stream));
    if (rcrit_host)
        CK(cudaMemcpyAsync(const_cast<double*>(ctx->rcrit), rcrit_host, (size_t)ctx->nb * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
    if (!a_is_current) ctx->a_valid = false;
    mo_status s = mo_step(ctx, dt, nsteps, nullptr);
    if (s != MO_OK) return s;
    CK(cudaMemcpyAsync(x_host, ctx->x, bytes, cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaMemcpyAsync(v_host, ctx->v, bytes, cudaMemcpyDeviceToHost, ctx->stream));
    mo_stats st;
    mo_status rs = status_from_stats(ctx, &st);
    if (rs == MO_ECUDA) return rs;
    if (stats_host) *stats_host = st;
    if (pairs_host && nsteps > 0) {
        long long n = st.nce_last;
        if (n > ctx->cap) n = ctx->cap;
        if (n > cap_host) n = cap_host;
        if (n > 0) {
            CK(cudaMemcpyAsync(pairs_host, ctx->pairs, (size_t)n * 2 * sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
            CK(cudaStreamSynchronize(ctx->stream));
        }
    }
    return rs;
}

extern "C" mo_status mo_accel_host(mo_ctx* ctx, const double* x_host, double* a_host) {
    if (!ctx || !x_host || !a_host) return MO_EINVAL;
    const size_t bytes = 3 * (size_t)ctx->ld * sizeof(double);
    CK(cudaMemcpyAsync(ctx->x, x_host, bytes, cudaMemcpyHostToDevice, ctx->stream));
    mo_status s = mo_accel(ctx);
    if (s != MO_OK) return s;
    CK(cudaMemcpyAsync(a_host, ctx->a, bytes, cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return MO_OK;
}

extern "C" mo_status mo_probe_fp64_peak(void* cuda_stream, int32_t reps, double* tflops_out, double* ms_out,
                                        double* tflops_mean_out) {
    if (!tflops_out || reps < 1) return MO_EINVAL;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    int dev = 0, nsm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        cudaGetLastError();
        return MO_ECUDA;
    }
    const int blocks = nsm * 8, threads = 256, iters = 1 << 14;
    double* buf = nullptr;
    if (cudaMalloc(reinterpret_cast<void**>(&buf), (size_t)blocks * threads * sizeof(double)) != cudaSuccess) {
        cudaGetLastError();
        return MO_ENOMEM;
    }
    cudaEvent_t e0, e1, ea, eb;
    cudaEventCreate(&e0); cudaEventCreate(&e1); cudaEventCreate(&ea); cudaEventCreate(&eb);
    double best = 1e300;
    mo_status rs = MO_OK;
    for (int r = 0; r < reps + 2; ++r) {  // two warm-ups
        if (r == 2) cudaEventRecord(ea, st);
        cudaEventRecord(e0, st);
        dfma_probe_kernel<<<blocks, threads, 0, st>>>(buf, iters, 0.999999, 1e-9);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) { rs = MO_ECUDA; break; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (r >= 2 && ms < best) best = ms;
    }
    float tot = 0.f;
    if (rs == MO_OK) {
        cudaEventRecord(eb, st);
        if (cudaEventSynchronize(eb) != cudaSuccess) rs = MO_ECUDA;
        else cudaEventElapsedTime(&tot, ea, eb);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaEventDestroy(ea); cudaEventDestroy(eb);
    cudaFree(buf);
    if (rs != MO_OK) { cudaGetLastError(); return rs; }
    const double flops = (double)blocks * threads * (double)iters * 32.0 * 2.0;
    *tflops_out = flops / (best * 1e-3) / 1e12;
    if (ms_out) *ms_out = best;
    if (tflops_mean_out) *tflops_mean_out = flops * reps / (tot * 1e-3) / 1e12;
    return MO_OK;
}

// ---- mo_accel_static: the pair accelerations of a small system with NO allocation anywhere ------------------------
// For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
// it): the same kernels as mo_accel takes for a mid-size system - pack_kernel<false, true>, pair_sym_kernel<2>,
// sym_reduce_kernel<false, false> - with their scratch (the packed j tiles, the work-unit list, the row and column
// partial sums) in ONE file-scope device array of fixed size instead of a context's cudaMalloc'ed buffers.  No context:
// the caller passes inputs and outputs.  Every GPU that loads the library holds the array (2.7 MB) until exit.
constexpr int STATIC_MAX_NB = 4096;                                      // mo_accel_static_max_nb()
constexpr int ST_IPT = 2;                                                // bodies per lane: the mid-size instance
constexpr int ST_R = sym_rows(ST_IPT);                                   // 256 rows per row block
constexpr int ST_NT = STATIC_MAX_NB / TJ;                                // 32 tiles
constexpr int ST_NI = (STATIC_MAX_NB + ST_R - 1) / ST_R;                 // 16 row blocks
constexpr int ST_NU = ST_NI * ST_NT - ST_IPT * (ST_NI * (ST_NI - 1) / 2);   // 272 units: one per (row block, j tile from its diagonal on)
constexpr size_t st_up(size_t b) { return (b + 255) & ~(size_t)255; }
constexpr size_t ST_OFF_TILES = 0;
constexpr size_t ST_OFF_UNITS = ST_OFF_TILES + st_up((size_t)ST_NT * SYM_TILE_BYTES);
constexpr size_t ST_OFF_USTART = ST_OFF_UNITS + st_up((size_t)ST_NU * sizeof(int4));
constexpr size_t ST_OFF_PARTI = ST_OFF_USTART + st_up((size_t)(ST_NI + 1) * sizeof(int));
constexpr size_t ST_OFF_PARTJ = ST_OFF_PARTI + st_up((size_t)ST_NU * 3 * ST_R * sizeof(double));
constexpr size_t ST_BYTES = ST_OFF_PARTJ + st_up((size_t)(3LL * ((long long)ST_NI * STATIC_MAX_NB - (long long)ST_R * (ST_NI * (ST_NI - 1) / 2))) * sizeof(double));
static_assert(STATIC_MAX_NB % ST_R == 0 && ST_BYTES < (3u << 20), "mo_accel_static: scratch layout");

// The scratch itself.  In HOST code this name is a host-side stand-in, not a device address: the kernels get the address
// cudaGetSymbolAddress returns (static_scratch_ptr below), never the name.
static __device__ __align__(256) unsigned char g_static_scratch[ST_BYTES];

// the work-unit list of this nb, written on the device (no host staging buffer): unit (I, t) = j tile t >= I * IPT of
// row block I, all four groups of 32 columns; ustart[I] = first unit of row block I
__global__ void static_plan_kernel(int4* __restrict__ units, int* __restrict__ ustart, int nI, int nTiles) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k <= nI) {
        // row blocks I' < k hold nTiles - I' * IPT units each (k = nI: the total)
        ustart[k] = k * nTiles - ST_IPT * (k * (k - 1) / 2);
    }
    if (k >= nI * nTiles) return;
    const int I = k / nTiles, t = k - I * nTiles;
    if (t < I * ST_IPT) return;
    const int u0 = I * nTiles - ST_IPT * (I * (I - 1) / 2);
    units[u0 + t - I * ST_IPT] = make_int4(I, t, t + 1, (TJ / 32) << 8);
}

// device address of the scratch on the CURRENT device: looked up once per device, with that device current
static cudaError_t static_scratch_ptr(unsigned char** out) {
    constexpr int MAXDEV = 64;
    static unsigned char* ptrs[MAXDEV] = {};
    static std::mutex mu;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= MAXDEV) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mu);
    if (!ptrs[dev]) {
        unsigned char* p = nullptr;
        e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_static_scratch);
        if (e != cudaSuccess) return e;
        if (!p || (reinterpret_cast<uintptr_t>(p) & 255u)) return cudaErrorInvalidSymbol;
        ptrs[dev] = p;
    }
    *out = ptrs[dev];
    return cudaSuccess;
}

extern "C" int32_t mo_accel_static_max_nb(void) { return STATIC_MAX_NB; }

extern "C" mo_status mo_accel_static(int32_t nb, int32_t ld, const double* gm, const double* x, const double* rcrit,
                                     double* a, void* cuda_stream) {
    if (nb < 1 || ld < nb || (ld & 3) || !gm || !x || !rcrit || !a) return MO_EINVAL;
    if (!aligned16(gm) || !aligned16(x) || !aligned16(rcrit) || !aligned16(a)) return MO_EINVAL;
    if (nb > STATIC_MAX_NB) return MO_ELIMIT;                            // the scratch is fixed: no fallback to an allocation
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    unsigned char* base = nullptr;
    if (static_scratch_ptr(&base) != cudaSuccess) { cudaGetLastError(); return MO_ECUDA; }
    const int nTiles = (nb + TJ - 1) / TJ, nbPad = nTiles * TJ;
    const int nI = (nbPad + ST_R - 1) / ST_R;
    const int nU = nI * nTiles - ST_IPT * (nI * (nI - 1) / 2);
    unsigned char* tiles = base + ST_OFF_TILES;
    int4* units = reinterpret_cast<int4*>(base + ST_OFF_UNITS);
    int* ustart = reinterpret_cast<int*>(base + ST_OFF_USTART);
    double* partI = reinterpret_cast<double*>(base + ST_OFF_PARTI);
    double* partJ = reinterpret_cast<double*>(base + ST_OFF_PARTJ);
    // Nothing in the scratch has to start at zero: every entry the reduce kernel reads (one row partial per unit, one
    // column partial per (row block, column at or right of its diagonal)) and every tile and unit record is rewritten
    // by this call before it is read, whatever the last call - of any nb - left there.
    const Gate open{nullptr, 0};
    static_plan_kernel<<<(nI * nTiles + 1 + 127) / 128, 128, 0, st>>>(units, ustart, nI, nTiles);
    pack_kernel<false, true><<<nTiles, TJ, 0, st>>>(const_cast<double*>(x), gm, rcrit, nb, nb, ld, tiles, nullptr, 0, 0.0, open);
    SymParams sp;
    sp.tiles = tiles; sp.x = x; sp.gm = gm; sp.rcrit = rcrit; sp.units = units; sp.partI = partI; sp.partJ = partJ;
    sp.nb = nb; sp.ld = ld; sp.nbPad = nbPad; sp.unit0 = 0; sp.gate = open;
    pair_sym_kernel<ST_IPT><<<nU, SYM_THREADS, 0, st>>>(sp);
    sym_reduce_kernel<false, false><<<dim3((nb + 31) / 32, 3), RED_THREADS, 0, st>>>(partI, partJ, ustart, nb, ld, nbPad, a, nullptr, 0.0,
                                                                                   0, nU, nullptr, ST_R, open);
    if (cudaGetLastError() != cudaSuccess) return MO_ECUDA;
    return MO_OK;
}
