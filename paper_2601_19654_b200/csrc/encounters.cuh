// encounters.cuh - close-encounter check (mce_snif).
//   boxes  (LOOP 1-2): per body, extremes of x and y over the step from the cubic Hermite
//                      interpolant through (x0, h v0) and (x1, h v1), padded by rcrit.
//   pairs  (LOOP 3)  : for i<j, boxes overlap in x and y AND the minimum over the step of
//                      the cubic Hermite interpolant of |x_i - x_j|^2 (interior minimum
//                      only when approaching at the start and receding at the end)
//                      is <= max(rcrit_i, rcrit_j)^2.
// The paper appends with an atomic capture in whatever order threads arrive
// (PAPER.md:264-269).  Here the list is deterministic and sorted by construction:
//   pass 1  thread-per-row i over TMA-staged tiles of j boxes counts the hits of each row,
//   scan    exclusive prefix sum of the row counts gives each row's slot range,
//   pass 2  one warp per non-empty row re-tests its j's in order and compacts the hits
//           with warp ballot + prefix popcounts straight into the row's slots.
// Both passes call the same pair test, written with explicit _rn intrinsics so that the
// compiler can neither contract nor reorder it: the two passes decide identically.
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

__device__ __forceinline__ bool box_gate(const double4& bi, const double2& ja, const double2& jb) {
    // {lox,hix} = ja, {loy,hiy} = jb of body j
    return (bi.x <= ja.y) & (ja.x <= bi.y) & (bi.z <= jb.y) & (jb.x <= bi.w);
}

// ---- O(N) kernel: boxes, and reset of the per-row counters and flags ------------------------
__global__ void __launch_bounds__(ON_BLOCK) boxes_kernel(EncState s, double4* __restrict__ box, int nbPad,
                                                         int* __restrict__ rowcnt, uint8_t* __restrict__ flag) {
    const int b = blockIdx.x * ON_BLOCK + threadIdx.x;
    if (b >= nbPad) return;
    double4 r;
    if (b < s.nb) {
        body_box(s.x0, s.v0, s.x1, s.v1, s.rcrit[b], s.ld, b, s.h, r);
        rowcnt[b] = 0;
        flag[b] = 0;
    } else {
        const double inf = __longlong_as_double(0x7ff0000000000000LL);
        r = make_double4(inf, -inf, inf, -inf);
    }
    box[b] = r;
}

// ---- pass 1: per-row hit counts ----------------------------------------------------------------
struct EncCountParams {
    EncState s;
    const double4* box;  // nbPad records
    int* rowcnt;
    int nTiles, tps;
};

__global__ void __launch_bounds__(CTA_THREADS) enc_count_kernel(EncCountParams p) {
    __shared__ __align__(128) unsigned char s_tiles[STAGES * BOX_TILE_BYTES];
    __shared__ __align__(8) uint64_t s_full[STAGES];
    __shared__ __align__(8) uint64_t s_empty[STAGES];

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    // rows of this CTA are [rb*TJ, rb*TJ+TJ): only tiles >= rb hold any j > i
    const int rb = blockIdx.x;
    const int t0 = max(blockIdx.y * p.tps, rb);
    const int t1 = min((blockIdx.y + 1) * p.tps, p.nTiles);
    const int nt = t1 - t0;
    if (nt <= 0) return;

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; ++s) { mbar_init(&s_full[s], 1); mbar_init(&s_empty[s], CONSUMER_THREADS / 32); }
        mbar_fence_init();
    }
    __syncthreads();

    if (warp == CONSUMER_THREADS / 32) {
        if (lane == 0) {
            const unsigned char* src = reinterpret_cast<const unsigned char*>(p.box) + (size_t)t0 * BOX_TILE_BYTES;
            for (int n = 0; n < nt; ++n) {
                const int st = n % STAGES;
                mbar_wait(&s_empty[st], ((n / STAGES) & 1) ^ 1);
                mbar_arrive_expect_tx(&s_full[st], BOX_TILE_BYTES);
                tma_load_1d(s_tiles + st * BOX_TILE_BYTES, src + (size_t)n * BOX_TILE_BYTES, BOX_TILE_BYTES, &s_full[st]);
            }
        }
        return;
    }

    const int i = rb * TJ + tid;
    const double inf = __longlong_as_double(0x7ff0000000000000LL);
    const double4 bi = (i < p.s.nb) ? p.box[i] : make_double4(inf, -inf, inf, -inf);
    int cnt = 0;
    for (int n = 0; n < nt; ++n) {
        const int st = n % STAGES;
        mbar_wait(&s_full[st], (n / STAGES) & 1);
        const double2* tj = reinterpret_cast<const double2*>(s_tiles + st * BOX_TILE_BYTES);
        const int j0 = (t0 + n) * TJ;
        const int jmin = (t0 + n == rb) ? (tid + 1) : 0;  // diagonal tile: j > i only
#pragma unroll 4
        for (int jj = 0; jj < TJ; ++jj) {
            const double2 ja = tj[2 * jj], jb = tj[2 * jj + 1];
            if (box_gate(bi, ja, jb) && jj >= jmin) cnt += pair_hit(p.s, i, j0 + jj) ? 1 : 0;
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&s_empty[st]);
    }
    if (cnt) atomicAdd(&p.rowcnt[i], cnt);
}

// ---- scan: rowoff = exclusive prefix sum of rowcnt; count -> stats ----------------------------
struct DevStats {
    long long steps_done, nce_last, nce_total;
    int drift_fail, max_newton;
    int overflow;  // sticky: some pass found more pairs than cap
    int pad;
};

constexpr int SCAN_THREADS = 1024;
__global__ void __launch_bounds__(SCAN_THREADS) enc_scan_kernel(const int* __restrict__ rowcnt, long long* __restrict__ rowoff,
                                                                int nb, long long cap, int step_inc, DevStats* __restrict__ st) {
    __shared__ long long wsum[SCAN_THREADS / 32];
    const int per = (nb + SCAN_THREADS - 1) / SCAN_THREADS;
    const int b0 = threadIdx.x * per, b1 = min(b0 + per, nb);
    long long local = 0;
    for (int b = b0; b < b1; ++b) local += rowcnt[b];
    long long incl = local;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        long long t = __shfl_up_sync(0xffffffffu, incl, o);
        if ((threadIdx.x & 31) >= o) incl += t;
    }
    if ((threadIdx.x & 31) == 31) wsum[threadIdx.x >> 5] = incl;
    __syncthreads();
    if (threadIdx.x < 32) {
        long long v = wsum[threadIdx.x], inc2 = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            long long t = __shfl_up_sync(0xffffffffu, inc2, o);
            if (threadIdx.x >= o) inc2 += t;
        }
        wsum[threadIdx.x] = inc2 - v;  // exclusive warp offsets
        if (threadIdx.x == 31) {
            st->nce_last = inc2;
            st->nce_total += inc2;
            st->steps_done += step_inc;
            if (inc2 > cap) st->overflow = 1;
        }
    }
    __syncthreads();
    long long run = wsum[threadIdx.x >> 5] + (incl - local);
    for (int b = b0; b < b1; ++b) { rowoff[b] = run; run += rowcnt[b]; }
}

// ---- pass 2: one warp per non-empty row, ballot + prefix compaction into the row's slots ----
struct EncWriteParams {
    EncState s;
    const double4* box;
    const int* rowcnt;
    const long long* rowoff;
    int* pairs;
    long long cap;
    uint8_t* flag;
};

__global__ void __launch_bounds__(256) enc_write_kernel(EncWriteParams p) {
    const int lane = threadIdx.x & 31;
    const int gw = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int nw = (gridDim.x * blockDim.x) >> 5;
    for (int row = gw; row < p.s.nb; row += nw) {
        const int cnt = p.rowcnt[row];
        if (cnt == 0) continue;
        const long long off = p.rowoff[row];
        const double4 bi = p.box[row];
        int written = 0;
        for (int j0 = (row + 1) & ~31; j0 < p.s.nb && written < cnt; j0 += 32) {
            const int j = j0 + lane;
            bool hit = false;
            if (j > row && j < p.s.nb) {
                const double4 bj = p.box[j];
                if (box_gate(bi, make_double2(bj.x, bj.y), make_double2(bj.z, bj.w))) hit = pair_hit(p.s, row, j);
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
