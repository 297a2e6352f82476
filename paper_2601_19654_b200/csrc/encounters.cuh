// encounters.cuh - close-encounter check (mce_snif).
//   boxes  (LOOP 1-2): per body, extremes of x and y over the step from the cubic Hermite
//                      interpolant through (x0, h v0) and (x1, h v1), padded by rcrit.
//   pairs  (LOOP 3)  : for i<j, boxes overlap in x and y AND the minimum over the step of
//                      the cubic Hermite interpolant of |x_i - x_j|^2 (interior minimum
//                      only when approaching at the start and receding at the end)
//                      is <= max(rcrit_i, rcrit_j)^2.
// The paper appends with an atomic capture in whatever order threads arrive
// (PAPER.md:264-269).  Here the list is deterministic and sorted:
//   sort    (performance only, never decides anything) bodies are binned on a 64 x 64 grid over
//           the bounding square of the boxes' lower corners, in Morton order of the cell, by a
//           counting sort (enc_key_kernel, enc_sortscatter_kernel); enc_tilebox_kernel takes the
//           bounding box of every run of TJ = 128 sorted boxes.  A row tile then only visits
//           the column tiles whose bounding box overlaps its own: the all-pairs gate of LOOP 3
//           is evaluated on ~1e7..1e8 instead of N^2/2 pairs, and skipped pairs are exactly
//           pairs the box gate rejects (the bounding boxes contain the boxes), so the flagged
//           set is unchanged.  The order inside a cell depends on atomics; nothing downstream
//           does (hits are ranked into sorted order).
//   find    thread-per-row i over TMA-staged tiles of j boxes.  The gate runs on
//           FP32 copies of the boxes rounded OUTWARD (lo down, hi up), so it can only pass
//           more pairs than the FP64 gate, never fewer; it costs 1 LDS.128 + 4 FSETP per
//           pair on the FP32/ALU pipes.  Survivors (~1e-5..1e-3 of the pairs) are compacted
//           per warp with ballot + prefix popcounts into a shared-memory queue and taken 32
//           at a time - one survivor per lane - through the exact FP64 box gate and the
//           exact pair test.  Hits bump their row's counter and go to an unsorted hit list.
//   scan    exclusive prefix sum of the row counts gives each row's slot range, the total
//           count and the overflow flag.
//   place   every hit drops its j into its row's slot range (scratch), then ranks itself
//           among its row's j's and writes (i, j) at rowoff[i] + rank: the final list is
//           sorted by (i, j) whatever order the atomics ran in.
//   overflow (count > cap): the list must hold the FIRST cap pairs in sorted order, which an
//           unsorted hit list cannot give; enc_write_kernel then re-tests the non-empty rows
//           in order (one warp per row, ballot compaction straight into the row's slots).
//           It exits at once when there was no overflow.
// The pair test is written with explicit _rn intrinsics so that the compiler can neither
// contract nor reorder it: every pass decides identically.
#pragma once
#include "common.cuh"

namespace mopal {

// ---- boxes ---------------------------------------------------------------------------
__device__ __forceinline__ void box_1d(double p0, double p1, double w0, double w1, double h, double& lo,
                                       double& hi) {
    double l = fmin(p0, p1), u = fmax(p0, p1);
    if (__dmul_rn(w0, w1) < 0.0) {
        const double k1 = __dmul_rn(h, w0);
        // k2 = -3 p0 - 2 h w0 + 3 p1 - h w1 ;  k3 = 2 p0 + h w0 - 2 p1 + h w1   (left to right)
        const double hw1 = __dmul_rn(h, w1);
        const double k2 = __dsub_rn(__dadd_rn(__dsub_rn(__dmul_rn(-3.0, p0), __dmul_rn(__dmul_rn(2.0, h), w0)),
                                              __dmul_rn(3.0, p1)), hw1);
        const double k3 = __dadd_rn(__dsub_rn(__dadd_rn(__dmul_rn(2.0, p0), k1), __dmul_rn(2.0, p1)), hw1);
        const double D = __dsub_rn(__dmul_rn(k2, k2), __dmul_rn(__dmul_rn(3.0, k3), k1));
        if (D >= 0.0) {
            const double sq = __dsqrt_rn(D);
            const double qq = (k2 >= 0.0) ? __dadd_rn(k2, sq) : __dsub_rn(k2, sq);
            if (qq != 0.0) {
                const double ta = __ddiv_rn(-k1, qq);
                if (ta > 0.0 && ta < 1.0) {
                    const double pp = __dadd_rn(__dmul_rn(__dadd_rn(__dmul_rn(__dadd_rn(__dmul_rn(k3, ta), k2), ta), k1), ta), p0);
                    l = fmin(l, pp); u = fmax(u, pp);
                }
            }
            if (k3 != 0.0) {
                const double tb = __ddiv_rn(-qq, __dmul_rn(3.0, k3));
                if (tb > 0.0 && tb < 1.0) {
                    const double pp = __dadd_rn(__dmul_rn(__dadd_rn(__dmul_rn(__dadd_rn(__dmul_rn(k3, tb), k2), tb), k1), tb), p0);
                    l = fmin(l, pp); u = fmax(u, pp);
                }
            }
        }
    }
    lo = l; hi = u;
}

// box record {lox, hix, loy, hiy}; pad records can never overlap anything
__device__ __forceinline__ void body_box(const double* __restrict__ x0, const double* __restrict__ v0,
                                         const double* __restrict__ x1, const double* __restrict__ v1,
                                         double rc, int ld, int b, double h, double4& out) {
    double lo, hi;
    box_1d(x0[b], x1[b], v0[b], v1[b], h, lo, hi);
    out.x = __dsub_rn(lo, rc); out.y = __dadd_rn(hi, rc);
    box_1d(x0[ld + b], x1[ld + b], v0[ld + b], v1[ld + b], h, lo, hi);
    out.z = __dsub_rn(lo, rc); out.w = __dadd_rn(hi, rc);
}

struct EncState {
    const double *x0, *v0, *x1, *v1, *rcrit;
    int nb, ld;
    int nbig;   // bodies 0..nbig-1 are big: padded boxes (LOOP 2), first members of pairs
                // (LOOP 3 `do i = 2, nbig`); nbig = nb: every body
    double h;
};

// ---- exact pair test (mce_min + threshold), identical operation order in both passes ----
__device__ __noinline__ bool pair_hit(const EncState& s, int i, int j) {
    double d0 = 0.0, d1 = 0.0, s0 = 0.0, s1 = 0.0;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const size_t o = (size_t)c * s.ld;
        const double D0 = __dsub_rn(s.x0[o + i], s.x0[o + j]);
        const double D1 = __dsub_rn(s.x1[o + i], s.x1[o + j]);
        const double U0 = __dsub_rn(s.v0[o + i], s.v0[o + j]);
        const double U1 = __dsub_rn(s.v1[o + i], s.v1[o + j]);
        d0 = __dadd_rn(d0, __dmul_rn(D0, D0));
        d1 = __dadd_rn(d1, __dmul_rn(D1, D1));
        s0 = __dadd_rn(s0, __dmul_rn(D0, U0));
        s1 = __dadd_rn(s1, __dmul_rn(D1, U1));
    }
    const double h = s.h;
    const double d0t = __dmul_rn(2.0, s0), d1t = __dmul_rn(2.0, s1);
    double d2min;
    if (__dmul_rn(d0t, h) <= 0.0 && __dmul_rn(d1t, h) >= 0.0) {
        const double c1 = __dmul_rn(h, d0t);
        const double hd1t = __dmul_rn(h, d1t);
        const double c2 = __dsub_rn(__dadd_rn(__dsub_rn(__dmul_rn(-3.0, d0), __dmul_rn(__dmul_rn(2.0, h), d0t)),
                                              __dmul_rn(3.0, d1)), hd1t);
        const double c3 = __dadd_rn(__dsub_rn(__dadd_rn(__dmul_rn(2.0, d0), c1), __dmul_rn(2.0, d1)), hd1t);
        const double D = fmax(__dsub_rn(__dmul_rn(c2, c2), __dmul_rn(__dmul_rn(3.0, c3), c1)), 0.0);
        const double den = __dadd_rn(c2, __dsqrt_rn(D));
        double tau = (den > 0.0) ? __ddiv_rn(-c1, den) : 0.0;
        tau = fmin(fmax(tau, 0.0), 1.0);
        d2min = fmax(__dadd_rn(__dmul_rn(__dadd_rn(__dmul_rn(__dadd_rn(__dmul_rn(c3, tau), c2), tau), c1), tau), d0), 0.0);
        d2min = fmin(d2min, fmin(d0, d1));
    } else {
        d2min = fmin(d0, d1);
    }
    const double rc = fmax(s.rcrit[i], s.rcrit[j]);
    return d2min <= __dmul_rn(rc, rc);
}

// conservative FP32 copy of a box: lo rounded down, hi rounded up
__device__ __forceinline__ float4 box_f32(const double4& b) {
    return make_float4(__double2float_rd(b.x), __double2float_ru(b.y), __double2float_rd(b.z), __double2float_ru(b.w));
}
__device__ __forceinline__ double4 pad_box() {   // can never overlap anything
    const double inf = __longlong_as_double(0x7ff0000000000000LL);
    return make_double4(inf, -inf, inf, -inf);
}
__device__ __forceinline__ float4 pad_boxf() {
    const float inf = __int_as_float(0x7f800000);
    return make_float4(inf, -inf, inf, -inf);
}

// per-pass device scratch of the encounter pipeline
struct EncBuf {
    double4* box;        // nbPad exact boxes {lox, hix, loy, hiy}
    float4* boxf;        // nbPad outward-rounded FP32 boxes (the j tiles of the find pass)
    int* rowcnt;         // nbPad hits per row
    int* rowfill;        // nbPad placement cursor per row
    long long* rowoff;   // nbPad exclusive prefix of rowcnt
    int2* hits;          // cap unsorted hits (i, j)
    int* tmpj;           // cap j's grouped by row, unsorted inside a row
    unsigned long long* nhit;  // hits appended this pass (may exceed cap)
    int* ovf_now;        // this pass found more pairs than cap
    int* nlong;          // rows with more than ENC_RANK_LONG hits this pass ...
    int* longrows;       // ... and their indices (any order), written by the scan
    // spatial ordering of this pass (performance only)
    float4* bpart;       // per block of the boxes kernel: {min lox, max lox, min loy, max loy}
    int* cellcnt;        // ENC_NCELL bodies per grid cell
    int* cellfill;       // ENC_NCELL placement cursors
    int* key;            // nbPad cell of each body
    int* perm;           // nbPad sorted position -> body
    float4* sboxf;       // nbPad FP32 boxes in sorted order (pad records at the end)
    float4* tbox;        // nTiles bounding box of each run of TJ sorted boxes
    int* tilecnt;        // nTiles hits per run of TJ rows (body order), the scan's block bases
    int* tbig;           // nTiles: 1 iff the run of TJ sorted boxes holds a big body (index < nbig)
};

constexpr int ENC_RANK_LONG = 64;                  // rows with more hits are ranked by whole CTAs
constexpr int ENC_GRID = 64;                       // cells per axis
constexpr int ENC_NCELL = ENC_GRID * ENC_GRID;

// block partial of the bounds of the boxes' lower corners (real bodies only) and reset of the
// cell counters; called by every thread of a boxes kernel (blocks of ON_BLOCK threads)
__device__ __forceinline__ void enc_bounds_partial(const EncBuf& e, bool real, const float4& bf, float4* sh4,
                                                   int nTiles) {
    const float inf = __int_as_float(0x7f800000);
    float mnx = real ? bf.x : inf, mxx = real ? bf.x : -inf, mny = real ? bf.z : inf, mxy = real ? bf.z : -inf;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        mnx = fminf(mnx, __shfl_down_sync(0xffffffffu, mnx, o));
        mxx = fmaxf(mxx, __shfl_down_sync(0xffffffffu, mxx, o));
        mny = fminf(mny, __shfl_down_sync(0xffffffffu, mny, o));
        mxy = fmaxf(mxy, __shfl_down_sync(0xffffffffu, mxy, o));
    }
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) sh4[w] = make_float4(mnx, mxx, mny, mxy);
    __syncthreads();
    if (threadIdx.x == 0) {
        float4 r = sh4[0];
#pragma unroll
        for (int k = 1; k < ON_BLOCK / 32; ++k) {
            r.x = fminf(r.x, sh4[k].x); r.y = fmaxf(r.y, sh4[k].y); r.z = fminf(r.z, sh4[k].z); r.w = fmaxf(r.w, sh4[k].w);
        }
        e.bpart[blockIdx.x] = r;
    }
    for (int c = blockIdx.x * ON_BLOCK + threadIdx.x; c < ENC_NCELL; c += gridDim.x * ON_BLOCK) {
        e.cellcnt[c] = 0; e.cellfill[c] = 0;
    }
    for (int c = blockIdx.x * ON_BLOCK + threadIdx.x; c < nTiles; c += gridDim.x * ON_BLOCK) e.tilecnt[c] = 0;
}

// ---- O(N) kernel: boxes, and reset of the per-row counters and flags ------------------------
__global__ void __launch_bounds__(ON_BLOCK) boxes_kernel(EncState s, EncBuf e, int nbPad, uint8_t* __restrict__ flag) {
    __shared__ float4 sh4[ON_BLOCK / 32];
    const int b = blockIdx.x * ON_BLOCK + threadIdx.x;
    if (b == 0) { *e.nhit = 0ull; *e.nlong = 0; }
    float4 bf = pad_boxf();
    if (b < nbPad) {
        double4 r;
        if (b < s.nb) {
            body_box(s.x0, s.v0, s.x1, s.v1, b < s.nbig ? s.rcrit[b] : 0.0, s.ld, b, s.h, r);
            flag[b] = 0;
            bf = box_f32(r);
        } else {
            r = pad_box();
        }
        e.boxf[b] = bf;
        e.rowcnt[b] = 0;
        e.rowfill[b] = 0;
        e.box[b] = r;
    }
    enc_bounds_partial(e, b < s.nb, bf, sh4, nbPad / TJ);
}

// ---- spatial ordering (performance only) ------------------------------------------------------
__device__ __forceinline__ unsigned spread6(unsigned v) {   // abcdef -> 0a0b0c0d0e0f
    v &= 0x3Fu;
    v = (v | (v << 4)) & 0x30Fu;   // ab....cdef  -> 0b11_0000_1111
    v = (v | (v << 2)) & 0x333u;   // 0b0011_0011_0011
    v = (v | (v << 1)) & 0x555u;   // 0b0101_0101_0101
    return v;
}

// cell of every body's lower box corner on the ENC_GRID^2 grid over the global bounds; histogram
__global__ void __launch_bounds__(ON_BLOCK) enc_key_kernel(EncBuf e, int nb, int nbPad, int npart) {
    __shared__ float4 sh4[ON_BLOCK / 32];
    __shared__ float4 bounds;
    const float inf = __int_as_float(0x7f800000);
    float4 r = make_float4(inf, -inf, inf, -inf);
    for (int k = threadIdx.x; k < npart; k += ON_BLOCK) {
        const float4 q = e.bpart[k];
        r.x = fminf(r.x, q.x); r.y = fmaxf(r.y, q.y); r.z = fminf(r.z, q.z); r.w = fmaxf(r.w, q.w);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        r.x = fminf(r.x, __shfl_down_sync(0xffffffffu, r.x, o));
        r.y = fmaxf(r.y, __shfl_down_sync(0xffffffffu, r.y, o));
        r.z = fminf(r.z, __shfl_down_sync(0xffffffffu, r.z, o));
        r.w = fmaxf(r.w, __shfl_down_sync(0xffffffffu, r.w, o));
    }
    if ((threadIdx.x & 31) == 0) sh4[threadIdx.x >> 5] = r;
    __syncthreads();
    if (threadIdx.x == 0) {
        float4 t = sh4[0];
#pragma unroll
        for (int k = 1; k < ON_BLOCK / 32; ++k) {
            t.x = fminf(t.x, sh4[k].x); t.y = fmaxf(t.y, sh4[k].y); t.z = fminf(t.z, sh4[k].z); t.w = fmaxf(t.w, sh4[k].w);
        }
        bounds = t;
    }
    __syncthreads();
    const int b = blockIdx.x * ON_BLOCK + threadIdx.x;
    if (b >= nbPad) return;
    int key = ENC_NCELL - 1;                 // pad records: last cell (they are placed after the bodies anyway)
    if (b < nb) {
        const float4 bf = e.boxf[b];
        const float wx = bounds.y - bounds.x, wy = bounds.w - bounds.z;
        const float sx = wx > 0.f ? (float)ENC_GRID / wx : 0.f, sy = wy > 0.f ? (float)ENC_GRID / wy : 0.f;
        // NaN / inf coordinates fall into cell 0 or the last cell: any cell is a valid choice
        int cx = (int)fminf(fmaxf((bf.x - bounds.x) * sx, 0.f), (float)(ENC_GRID - 1));
        int cy = (int)fminf(fmaxf((bf.z - bounds.z) * sy, 0.f), (float)(ENC_GRID - 1));
        cx = min(max(cx, 0), ENC_GRID - 1); cy = min(max(cy, 0), ENC_GRID - 1);
        key = (int)(spread6((unsigned)cx) | (spread6((unsigned)cy) << 1));
        atomicAdd(&e.cellcnt[key], 1);
    }
    e.key[b] = key;
}

// counting sort: every block prefix-sums the ENC_NCELL counters itself, then places its bodies
__global__ void __launch_bounds__(ON_BLOCK) enc_sortscatter_kernel(EncBuf e, int nb, int nbPad) {
    __shared__ int off[ENC_NCELL];
    __shared__ int wtot[ON_BLOCK / 32];
    constexpr int PER = ENC_NCELL / ON_BLOCK;   // 16 consecutive cells per thread
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    int c[PER], loc = 0;
#pragma unroll
    for (int k = 0; k < PER; ++k) { c[k] = e.cellcnt[tid * PER + k]; loc += c[k]; }
    int incl = loc;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    if (lane == 31) wtot[warp] = incl;
    __syncthreads();
    int wbase = 0;
#pragma unroll
    for (int k = 0; k < ON_BLOCK / 32; ++k) wbase += (k < warp) ? wtot[k] : 0;
    int run = wbase + incl - loc;
#pragma unroll
    for (int k = 0; k < PER; ++k) { off[tid * PER + k] = run; run += c[k]; }
    __syncthreads();
    const int b = blockIdx.x * ON_BLOCK + tid;
    if (b >= nbPad) return;
    if (b < nb) {
        const int key = e.key[b];
        const int pos = off[key] + atomicAdd(&e.cellfill[key], 1);
        e.perm[pos] = b;
        e.sboxf[pos] = e.boxf[b];
    } else {                                    // pad records keep their place at the end
        e.perm[b] = b;
        e.sboxf[b] = pad_boxf();
    }
}

// bounding box of each run of TJ sorted boxes, and whether the run holds a big body: a pair of
// runs without one has no pair whose first member is big (LOOP 3 `do i = 2, nbig`)
__global__ void __launch_bounds__(TJ) enc_tilebox_kernel(EncBuf e, int nbig) {
    __shared__ float4 sh4[TJ / 32];
    float4 r = e.sboxf[blockIdx.x * TJ + threadIdx.x];    // {lox, hix, loy, hiy}; pads are (+inf, -inf, ..)
    const int big = __syncthreads_or(e.perm[blockIdx.x * TJ + threadIdx.x] < nbig);
    if (threadIdx.x == 0) e.tbig[blockIdx.x] = big ? 1 : 0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        r.x = fminf(r.x, __shfl_down_sync(0xffffffffu, r.x, o));
        r.y = fmaxf(r.y, __shfl_down_sync(0xffffffffu, r.y, o));
        r.z = fminf(r.z, __shfl_down_sync(0xffffffffu, r.z, o));
        r.w = fmaxf(r.w, __shfl_down_sync(0xffffffffu, r.w, o));
    }
    if ((threadIdx.x & 31) == 0) sh4[threadIdx.x >> 5] = r;
    __syncthreads();
    if (threadIdx.x == 0) {
        float4 t = sh4[0];
#pragma unroll
        for (int k = 1; k < TJ / 32; ++k) {
            t.x = fminf(t.x, sh4[k].x); t.y = fmaxf(t.y, sh4[k].y); t.z = fminf(t.z, sh4[k].z); t.w = fmaxf(t.w, sh4[k].w);
        }
        e.tbox[blockIdx.x] = t;
    }
}

// ---- find: FP32 gate over the pairs of overlapping tiles, exact test on the survivors ---------
constexpr int BOXF_TILE_BYTES = TJ * 16;   // TJ x float4
constexpr int ENC_BATCH = 8;               // j's gated between two survivor checks
constexpr int ENC_QCAP = 64;               // per-warp survivor queue (a drain leaves < 32)
constexpr int ENC_UNSORTED_TILES = 40;     // up to this many tiles (N <= 5120) the find pass runs without the spatial ordering
constexpr int ENC_WIN = 1024;              // column tiles examined per window (candidate list in smem)

struct EncFindParams {
    EncState s;
    EncBuf e;
    long long cap;
    int nTiles;
    int unsorted;        // 1: no spatial ordering (a few tiles only: every pair of tiles is gated, in body order)
};

__device__ __forceinline__ bool gate_f32(const float4& a, const float4& b) {
    return (a.x <= b.y) & (b.x <= a.y) & (a.z <= b.w) & (b.z <= a.w);
}
__device__ __forceinline__ bool gate_f64(const double4& a, const double4& b) {
    return (a.x <= b.y) & (b.x <= a.y) & (a.z <= b.w) & (b.z <= a.w);
}

// exact FP64 gate and exact pair test of bodies i < j; a hit bumps its row's counters and goes to
// the unsorted hit list
__device__ __forceinline__ void enc_exact_body(const EncFindParams& p, int i, int j) {
    if (i >= p.s.nbig) return;                 // first member must be a big body
    const double4 bi = p.e.box[i], bj = p.e.box[j];
    if (!gate_f64(bi, bj)) return;
    if (!pair_hit(p.s, i, j)) return;
    atomicAdd(&p.e.rowcnt[i], 1);
    atomicAdd(&p.e.tilecnt[i / TJ], 1);
    const unsigned long long pos = atomicAdd(p.e.nhit, 1ull);
    if ((long long)pos < p.cap) p.e.hits[pos] = make_int2(i, j);
}

// one survivor per lane (sorted positions c.x < c.y): (i, j) = (smaller, larger) body index
__device__ __forceinline__ void enc_exact(const EncFindParams& p, int2 c) {
    const int ba = p.unsorted ? c.x : p.e.perm[c.x], bb = p.unsorted ? c.y : p.e.perm[c.y];
    enc_exact_body(p, min(ba, bb), max(ba, bb));
}

// ---- big x all find for few big bodies (`do i = 2, nbig` x `do j = i+1, nbod`
// with N_big <= ~100).  No spatial ordering: the nbig x nb rectangle of FP32 gates is
// small (1e8 at nb = 1e6, nbig = 100).  Every thread keeps BIGF_JPT bodies j (body order) in
// registers and sweeps the big boxes i < j, staged BIGF_CHUNK at a time in shared memory (one
// broadcast LDS.128 + 4 FSETP per gate); the rare survivors go straight through the exact test.
constexpr int BIGF_THREADS = 256;
constexpr int BIGF_JPT = 4;
constexpr int BIGF_CHUNK = 1024;
constexpr int BIGF_BATCH = 4;              // big boxes gated between two survivor checks
constexpr int BIGF_QCAP = 64;              // per-warp survivor queue (a drain leaves < 32)

__global__ void __launch_bounds__(BIGF_THREADS) enc_bigfind_kernel(EncFindParams p) {
    __shared__ float4 sbig[BIGF_CHUNK];
    __shared__ int2 s_q[BIGF_THREADS / 32][BIGF_QCAP];
    const int tid = threadIdx.x, lane = tid & 31;
    const unsigned full = 0xffffffffu, lt = (1u << lane) - 1u;
    const int jbase = blockIdx.x * (BIGF_THREADS * BIGF_JPT) + tid;
    float4 bj[BIGF_JPT];
#pragma unroll
    for (int k = 0; k < BIGF_JPT; ++k) {
        const int j = jbase + k * BIGF_THREADS;
        bj[k] = j < p.s.nb ? p.e.boxf[j] : pad_boxf();
    }
    int2* q = s_q[tid >> 5];
    int qhead = 0, qn = 0;                     // warp-uniform
    const int jmax = min(p.s.nb, (int)(blockIdx.x + 1) * (BIGF_THREADS * BIGF_JPT)) - 1;   // largest j of this CTA
    const int ilim = min(p.s.nbig, jmax);                                                  // rows i < j <= jmax
    for (int i0 = 0; i0 < ilim; i0 += BIGF_CHUNK) {
        const int n = min(BIGF_CHUNK, ilim - i0);
        const int npad = (n + BIGF_BATCH - 1) / BIGF_BATCH * BIGF_BATCH;
        __syncthreads();
        for (int t = tid; t < npad; t += BIGF_THREADS) sbig[t] = t < n ? p.e.boxf[i0 + t] : pad_boxf();
        __syncthreads();
#pragma unroll 1
        for (int ii = 0; ii < npad; ii += BIGF_BATCH) {
            bool any = false;
#pragma unroll
            for (int u = 0; u < BIGF_BATCH; ++u) {
                const float4 bi = sbig[ii + u];
#pragma unroll
                for (int k = 0; k < BIGF_JPT; ++k) any |= gate_f32(bi, bj[k]);
            }
            if (__any_sync(full, any)) {       // some lane has a survivor in this batch
#pragma unroll 1
                for (int u = 0; u < BIGF_BATCH; ++u) {
                    const float4 bi = sbig[ii + u];
                    const int i = i0 + ii + u;
#pragma unroll
                    for (int k = 0; k < BIGF_JPT; ++k) {
                        const int j = jbase + k * BIGF_THREADS;
                        const bool has = gate_f32(bi, bj[k]) && (i < j);
                        const unsigned bal = __ballot_sync(full, has);
                        if (bal == 0u) continue;
                        if (has) q[(qhead + qn + __popc(bal & lt)) & (BIGF_QCAP - 1)] = make_int2(i, j);
                        qn += __popc(bal);
                        __syncwarp();
                        if (qn >= 32) {        // a full warp of survivors through the exact test
                            const int2 c = q[(qhead + lane) & (BIGF_QCAP - 1)];
                            enc_exact_body(p, c.x, c.y);
                            qhead = (qhead + 32) & (BIGF_QCAP - 1);
                            qn -= 32;
                            __syncwarp();
                        }
                    }
                }
            }
        }
    }
    if (lane < qn) {
        const int2 c = q[(qhead + lane) & (BIGF_QCAP - 1)];
        enc_exact_body(p, c.x, c.y);
    }
}

// CTA (rb, y) owns the rb-th run of TJ sorted boxes (one per compute thread) and visits the column
// tiles t >= rb with (t - rb) % gridDim.y == y whose bounding box overlaps its own (the split over y
// spreads the rows of dense regions, which overlap many tiles, over several CTAs); a fifth warp
// streams those tiles (TMA).
__global__ void __launch_bounds__(CTA_THREADS) enc_find_kernel(EncFindParams p) {
    __shared__ __align__(128) unsigned char s_tiles[STAGES * BOXF_TILE_BYTES];
    __shared__ __align__(8) uint64_t s_full[STAGES];
    __shared__ __align__(8) uint64_t s_empty[STAGES];
    __shared__ int2 s_q[CONSUMER_THREADS / 32][ENC_QCAP];
    __shared__ int s_list[ENC_WIN];
    __shared__ int s_n;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int rb = blockIdx.x;
    const float4 own = p.unsorted ? make_float4(0.f, 0.f, 0.f, 0.f) : p.e.tbox[rb];   // (not used without the ordering)
    const bool rbig = p.unsorted ? rb * TJ < p.s.nbig : p.e.tbig[rb] != 0;
    const float4* __restrict__ boxes = p.unsorted ? p.e.boxf : p.e.sboxf;

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; ++s) { mbar_init(&s_full[s], 1); mbar_init(&s_empty[s], CONSUMER_THREADS / 32); }
        mbar_fence_init();
    }
    const unsigned full = 0xffffffffu, lt = (1u << lane) - 1u;
    const bool producer = warp == CONSUMER_THREADS / 32;
    const int si = rb * TJ + (producer ? 0 : tid);
    const float4 bi = boxes[si];              // pad records hold the never-overlapping box
    int2* q = s_q[producer ? 0 : warp];
    int qhead = 0, qn = 0;                    // warp-uniform
    int nglob = 0;                            // tiles streamed so far (ring position), CTA-uniform

    const int S = gridDim.y;
    for (int w0 = rb + blockIdx.y; w0 < p.nTiles; w0 += ENC_WIN * S) {
        __syncthreads();                      // previous window fully consumed (and the barriers initialised)
        if (tid == 0) s_n = 0;
        __syncthreads();
        for (int k = tid; k < ENC_WIN; k += CTA_THREADS) {
            const int t = w0 + k * S;
            if (t < p.nTiles && (p.unsorted ? rbig : gate_f32(own, p.e.tbox[t]) && (rbig || p.e.tbig[t] != 0))) s_list[atomicAdd(&s_n, 1)] = t;
        }
        __syncthreads();
        const int nt = s_n;

        if (producer) {  // ---- TMA producer warp ----
            if (lane == 0) {
                const unsigned char* src = reinterpret_cast<const unsigned char*>(boxes);
                for (int n = 0; n < nt; ++n) {
                    const int g = nglob + n, st = g % STAGES;
                    mbar_wait(&s_empty[st], ((g / STAGES) & 1) ^ 1);
                    mbar_arrive_expect_tx(&s_full[st], BOXF_TILE_BYTES);
                    tma_load_1d(s_tiles + st * BOXF_TILE_BYTES, src + (size_t)s_list[n] * BOXF_TILE_BYTES, BOXF_TILE_BYTES,
                                &s_full[st]);
                }
            }
        } else {
            for (int n = 0; n < nt; ++n) {
                const int g = nglob + n, st = g % STAGES;
                mbar_wait(&s_full[st], (g / STAGES) & 1);
                const float4* tj = reinterpret_cast<const float4*>(s_tiles + st * BOXF_TILE_BYTES);
                const int t = s_list[n];
                const int j0 = t * TJ;
                const int jmin = (t == rb) ? tid + 1 : 0;         // diagonal tile: sorted position j > i only
#pragma unroll 1
                for (int jj = 0; jj < TJ; jj += ENC_BATCH) {
                    bool any = false;
#pragma unroll
                    for (int u = 0; u < ENC_BATCH; ++u) any |= gate_f32(bi, tj[jj + u]);
                    if (__any_sync(full, any)) {                  // rare: some lane has a survivor in this batch
#pragma unroll 1
                        for (int u = 0; u < ENC_BATCH; ++u) {
                            const bool has = gate_f32(bi, tj[jj + u]) && (jj + u >= jmin);
                            const unsigned bal = __ballot_sync(full, has);
                            if (bal == 0u) continue;
                            if (has) q[(qhead + qn + __popc(bal & lt)) & (ENC_QCAP - 1)] = make_int2(si, j0 + jj + u);
                            qn += __popc(bal);
                            __syncwarp();
                            if (qn >= 32) {                       // a full warp of survivors
                                enc_exact(p, q[(qhead + lane) & (ENC_QCAP - 1)]);
                                qhead = (qhead + 32) & (ENC_QCAP - 1);
                                qn -= 32;
                                __syncwarp();
                            }
                        }
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&s_empty[st]);
            }
        }
        nglob += nt;
    }
    if (!producer && lane < qn) enc_exact(p, q[(qhead + lane) & (ENC_QCAP - 1)]);
}

// ---- scan: rowoff = exclusive prefix sum of rowcnt; count -> stats ----------------------------
struct DevStats {
    long long steps_done, nce_last, nce_total;
    int drift_fail, max_newton;
    int overflow;  // sticky: some pass found more pairs than cap
    int resolve_fail;  // cumulative: encounter components the Bulirsch-Stoer solve gave up on
};

// one block per run of TJ rows: the block's base is the sum of the per-tile hit counts before it
// (tilecnt, bumped next to rowcnt by the find pass), so every block scans only its own TJ counters
__global__ void __launch_bounds__(TJ) enc_scan_kernel(EncBuf e, int nTiles, long long cap, int step_inc,
                                                       DevStats* __restrict__ st) {
    __shared__ long long wpre[TJ / 32], wtot[TJ / 32];
    __shared__ int wrow[TJ / 32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, blk = blockIdx.x;
    long long pre = 0, tot = 0;
    for (int k = tid; k < nTiles; k += TJ) {
        const int c = e.tilecnt[k];
        pre += (k < blk) ? c : 0;
        tot += c;
    }
    const int c = e.rowcnt[blk * TJ + tid];
    int incl = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        pre += __shfl_down_sync(0xffffffffu, pre, o);
        tot += __shfl_down_sync(0xffffffffu, tot, o);
    }
    if (lane == 0) { wpre[warp] = pre; wtot[warp] = tot; }
    if (lane == 31) wrow[warp] = incl;
    __syncthreads();
    long long base = 0, total = 0;
    int wbase = 0;
#pragma unroll
    for (int k = 0; k < TJ / 32; ++k) {
        base += wpre[k]; total += wtot[k];
        wbase += (k < warp) ? wrow[k] : 0;
    }
    e.rowoff[blk * TJ + tid] = base + wbase + (incl - c);
    if (c > ENC_RANK_LONG && total <= cap) e.longrows[atomicAdd(e.nlong, 1)] = blk * TJ + tid;
    if (blk == 0 && tid == 0) {
        st->nce_last = total;
        st->nce_total += total;
        st->steps_done += step_inc;
        *e.ovf_now = total > cap ? 1 : 0;
        if (total > cap) st->overflow = 1;
    }
}

// ---- place: hits -> sorted list (no overflow) ------------------------------------------------
__global__ void __launch_bounds__(256) enc_scatter_kernel(EncBuf e, uint8_t* __restrict__ flag) {
    if (*e.ovf_now) return;
    const unsigned long long n = *e.nhit;
    for (unsigned long long h = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; h < n;
         h += (unsigned long long)gridDim.x * blockDim.x) {
        const int2 c = e.hits[h];
        const int k = atomicAdd(&e.rowfill[c.x], 1);
        e.tmpj[e.rowoff[c.x] + k] = c.y;
        flag[c.x] = 1;
        flag[c.y] = 1;
    }
}

// short rows (<= ENC_RANK_LONG hits): every hit ranks itself among the j's of its row.  Long rows
// (a giant planet's row holds thousands of hits; the scan listed them): the row's j's are dealt in
// blocks of 256 to CTAs, which stream the whole row through shared memory and count, per element,
// the smaller j's (4 compares per LDS.128).
constexpr int ENC_RANK_TILE = 2048;
__global__ void __launch_bounds__(256) enc_rank_kernel(EncBuf e, int* __restrict__ pairs) {
    __shared__ __align__(16) int s_key[ENC_RANK_TILE];
    if (*e.ovf_now) return;
    const unsigned long long n = *e.nhit;
    for (unsigned long long h = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; h < n;
         h += (unsigned long long)gridDim.x * blockDim.x) {
        const int2 c = e.hits[h];
        const int cnt = e.rowcnt[c.x];
        if (cnt > ENC_RANK_LONG) continue;
        const long long off = e.rowoff[c.x];
        const int* seg = e.tmpj + off;
        int rank = 0;
        for (int k = 0; k < cnt; ++k) rank += (seg[k] < c.y) ? 1 : 0;   // the j's of a row are distinct
        const long long pos = off + rank;
        pairs[2 * pos] = c.x;
        pairs[2 * pos + 1] = c.y;
    }
    const int nlong = *e.nlong;
    int ubase = 0;                                                       // units before this row (CTA-uniform)
    for (int L = 0; L < nlong; ++L) {
        const int row = e.longrows[L];
        const int cnt = e.rowcnt[row];
        const long long off = e.rowoff[row];
        const int* seg = e.tmpj + off;
        const int nblk = (cnt + 255) / 256;
        int u = ubase + ((int)blockIdx.x - ubase % (int)gridDim.x + (int)gridDim.x) % (int)gridDim.x;
        for (; u < ubase + nblk; u += gridDim.x) {
            const int k = (u - ubase) * 256 + threadIdx.x;
            const int j = k < cnt ? seg[k] : 0;
            int rank = 0;
            for (int t0 = 0; t0 < cnt; t0 += ENC_RANK_TILE) {
                __syncthreads();
                for (int q = threadIdx.x; q < ENC_RANK_TILE; q += 256) s_key[q] = (t0 + q < cnt) ? seg[t0 + q] : 0x7fffffff;
                __syncthreads();
                const int4* t4 = reinterpret_cast<const int4*>(s_key);
                const int lim = min(ENC_RANK_TILE, (cnt - t0 + 3) & ~3) / 4;
#pragma unroll 4
                for (int q = 0; q < lim; ++q) {
                    const int4 v = t4[q];
                    rank += (v.x < j) + (v.y < j) + (v.z < j) + (v.w < j);
                }
            }
            if (k < cnt) {
                pairs[2 * (off + rank)] = row;
                pairs[2 * (off + rank) + 1] = j;
            }
        }
        ubase += nblk;
    }
}

// ---- overflow fallback: one warp per non-empty row, in-order ballot compaction ---------------
struct EncWriteParams {
    EncState s;
    EncBuf e;
    int* pairs;
    long long cap;
    uint8_t* flag;
};

__global__ void __launch_bounds__(256) enc_write_kernel(EncWriteParams p) {
    if (*p.e.ovf_now == 0) return;
    const int lane = threadIdx.x & 31;
    const int gw = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int nw = (gridDim.x * blockDim.x) >> 5;
    for (int row = gw; row < p.s.nbig; row += nw) {
        const int cnt = p.e.rowcnt[row];
        if (cnt == 0) continue;
        const long long off = p.e.rowoff[row];
        const double4 bi = p.e.box[row];
        int written = 0;
        for (int j0 = (row + 1) & ~31; j0 < p.s.nb && written < cnt; j0 += 32) {
            const int j = j0 + lane;
            bool hit = false;
            if (j > row && j < p.s.nb) {
                if (gate_f64(bi, p.e.box[j])) hit = pair_hit(p.s, row, j);
            }
            const unsigned m = __ballot_sync(0xffffffffu, hit);
            if (hit) {
                const int rank = written + __popc(m & ((1u << lane) - 1u));
                const long long pos = off + rank;
                if (rank < cnt && pos < p.cap) { p.pairs[2 * pos] = row; p.pairs[2 * pos + 1] = j; }
                p.flag[j] = 1;
            }
            written += __popc(m);
        }
        if (lane == 0) p.flag[row] = 1;
    }
}

}  // namespace mopal
