// step_small.cuh - the whole pre-acceleration part of the hybrid step in ONE single-CTA kernel for
// nb <= 1024 bodies (the paper's own regime, N <= 1000, and BASELINE.json's config 0),
// where a step is launch-latency bound: 13 launches of a few microseconds each become 4.
//   [mce_hill] -> kick (LOOP 1) -> sum gm v (LOOP 2) -> jump (LOOP 3) -> x0, v0 copy
//   (LOOP 4) -> Kepler drift -> mce_snif boxes and pair test
//    -> sum gm v -> jump
// One thread per body, block-wide reductions and barriers only.  The arithmetic of every stage is the
// device function the multi-CTA kernels use (drift_body, box_1d, pair_hit, hill_body), so only the order
// of the two 3-vector reductions differs from the large-N path.
#pragma once
#include "glue.cuh"
#include "support.cuh"

namespace mopal {

constexpr int SMALL_MAX = 1024;
constexpr int SMALL_QCAP = 2048;      // box-gate survivors held in shared memory (more: row-per-thread fallback)

struct SmallParams {
    MidParams m;          // x, v, x0, v0, gm, rcrit, enc (box, boxf), flag, st, nb, ld, nbig, hj_over_mu, mu, h
    const double* a;
    double hk;
    int* pairs;
    long long cap;
    int hill_mode;        // -1: rcrit as given
    double hill_n;
};

__device__ __forceinline__ int block_excl_scan_1024(int v, int* sh, int& total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    if (lane == 31) sh[warp] = incl;
    __syncthreads();
    if (warp == 0) {
        int w = sh[lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, w, o);
            if (lane >= o) w += t;
        }
        sh[32 + lane] = w;      // inclusive over warps
    }
    __syncthreads();
    total = sh[32 + 31];
    return (warp ? sh[32 + warp - 1] : 0) + incl - v;
}

__global__ void __launch_bounds__(SMALL_MAX) step_small_kernel(SmallParams q) {
    __shared__ double sh3[SMALL_MAX / 32][3];
    __shared__ float4 s_boxf[SMALL_MAX];
    __shared__ int s_scan[64];
    __shared__ int s_rowcnt[SMALL_MAX];
    __shared__ int2 s_q[SMALL_QCAP];
    __shared__ int s_qn;
    const MidParams& p = q.m;
    const int b = threadIdx.x, ld = p.ld;
    // launched with just enough warps for nb bodies: the reductions below walk all 32 warp slots
    if (b < SMALL_MAX / 32) { sh3[b][0] = 0.0; sh3[b][1] = 0.0; sh3[b][2] = 0.0; }
    if (b < 64) s_scan[b] = 0;
    __syncthreads();
    const bool live = b < p.nb;
    double x = 0, y = 0, z = 0, vx = 0, vy = 0, vz = 0, g = 0;
    if (live) {
        x = p.x[b]; y = p.x[ld + b]; z = p.x[2 * ld + b];
        vx = p.v[b]; vy = p.v[ld + b]; vz = p.v[2 * ld + b];
        g = p.gm[b];
    }
    double rc = live ? p.rcrit[b] : 0.0;
    if (q.hill_mode >= 0) {     // mce_hill at the start of the step, from the state before the kick
        double P0 = 0, P1 = 0, P2 = 0;
        if (q.hill_mode == 1) {
            P0 = g * vx; P1 = g * vy; P2 = g * vz;
            block_sum3<SMALL_MAX>(P0, P1, P2, sh3);
            __syncthreads();
        }
        if (live) {
            rc = q.hill_n * hill_body(x, y, z, vx, vy, vz, g, p.mu, P0, P1, P2, q.hill_mode);
            const_cast<double*>(p.rcrit)[b] = rc;
        }
    }
    // kick, sum gm v, jump, snapshot
    if (live) { vx = fma(q.hk, q.a[b], vx); vy = fma(q.hk, q.a[ld + b], vy); vz = fma(q.hk, q.a[2 * ld + b], vz); }
    double P0 = g * vx, P1 = g * vy, P2 = g * vz;
    block_sum3<SMALL_MAX>(P0, P1, P2, sh3);
    __syncthreads();
    float4 bf = pad_boxf();
    double s0 = 0, s1 = 0, s2 = 0;
    if (live) {
        x += p.hj_over_mu * P0; y += p.hj_over_mu * P1; z += p.hj_over_mu * P2;
        p.x0[b] = x; p.x0[ld + b] = y; p.x0[2 * ld + b] = z;
        p.v0[b] = vx; p.v0[ld + b] = vy; p.v0[2 * ld + b] = vz;
        const double x0 = x, y0 = y, vx0 = vx, vy0 = vy;
        int iters;
        const int fail = drift_body(p.mu, p.h, x, y, z, vx, vy, vz, &iters);
        if (fail) atomicAdd(&p.st->drift_fail, 1);
        if (iters > 3) atomicMax(&p.st->max_newton, iters);
        p.x[b] = x; p.x[ld + b] = y; p.x[2 * ld + b] = z;          // x1: what the pair test reads
        p.v[b] = vx; p.v[ld + b] = vy; p.v[2 * ld + b] = vz;
        const double pad = b < p.nbig ? rc : 0.0;                    // LOOP 2 pads the big bodies only
        double lo, hi;
        double4 bx;
        box_1d(x0, x, vx0, vx, p.h, lo, hi);
        bx.x = __dsub_rn(lo, pad); bx.y = __dadd_rn(hi, pad);
        box_1d(y0, y, vy0, vy, p.h, lo, hi);
        bx.z = __dsub_rn(lo, pad); bx.w = __dadd_rn(hi, pad);
        p.enc.box[b] = bx;
        bf = box_f32(bx);
        p.flag[b] = 0;
        s0 = g * vx; s1 = g * vy; s2 = g * vz;
    }
    s_boxf[b] = bf;
    block_sum3<SMALL_MAX>(s0, s1, s2, sh3);      // its barriers also publish x1, v1, boxes and flags to the CTA
    __syncthreads();

    // mce_snif LOOP 3: rows i < nbig, j > i.  (A) every thread gates its row against the FP32 outward-rounded
    // boxes and queues the survivors; (B) the whole CTA takes the survivors through the exact FP64 gate and
    // the exact pair test, one per thread (a giant's row alone holds most of them); (C) row counts -> offsets;
    // (D) every hit ranks itself among its row's hits -> sorted list whatever order the queue filled in.
    EncState es;
    es.x0 = p.x0; es.v0 = p.v0; es.x1 = p.x; es.v1 = p.v; es.rcrit = p.rcrit;
    es.nb = p.nb; es.ld = ld; es.nbig = p.nbig; es.h = p.h;
    const bool row = live && b < p.nbig;
    s_rowcnt[b] = 0;
    if (b == 0) s_qn = 0;
    __syncthreads();
    if (row) {
        for (int j = b + 1; j < p.nb; ++j) {
            if (gate_f32(bf, s_boxf[j])) {
                const int k = atomicAdd(&s_qn, 1);
                if (k < SMALL_QCAP) s_q[k] = make_int2(b, j);
            }
        }
    }
    __syncthreads();
    const int nq = s_qn;
    int total;
    if (nq <= SMALL_QCAP) {
        for (int k = b; k < nq; k += blockDim.x) {
            const int2 c = s_q[k];
            if (gate_f64(p.enc.box[c.x], p.enc.box[c.y]) && pair_hit(es, c.x, c.y)) atomicAdd(&s_rowcnt[c.x], 1);
            else s_q[k].x = -1;                                        // not a hit
        }
        __syncthreads();
        const int cnt = s_rowcnt[b];
        const int off = block_excl_scan_1024(cnt, s_scan, total);
        __syncthreads();
        s_rowcnt[b] = off;                                             // now the row's offset
        __syncthreads();
        for (int k = b; k < nq; k += blockDim.x) {
            const int2 c = s_q[k];
            if (c.x < 0) continue;
            int rank = 0;
            for (int t = 0; t < nq; ++t) {
                const int2 o = s_q[t];
                rank += (o.x == c.x && o.y < c.y) ? 1 : 0;
            }
            const int pos = s_rowcnt[c.x] + rank;
            if (pos < q.cap) { q.pairs[2 * pos] = c.x; q.pairs[2 * pos + 1] = c.y; }
            p.flag[c.x] = 1;
            p.flag[c.y] = 1;
        }
    } else {
        // more survivors than the queue holds (huge rcrit): row per thread, count then write in order
        const double4 bi = row ? p.enc.box[b] : pad_box();
        int cnt = 0;
        if (row) {
            for (int j = b + 1; j < p.nb; ++j)
                if (gate_f32(bf, s_boxf[j]) && gate_f64(bi, p.enc.box[j]) && pair_hit(es, b, j)) ++cnt;
        }
        const int off = block_excl_scan_1024(cnt, s_scan, total);
        if (row && cnt > 0) {
            int k = off;
            for (int j = b + 1; j < p.nb && k < off + cnt; ++j) {
                if (gate_f32(bf, s_boxf[j]) && gate_f64(bi, p.enc.box[j]) && pair_hit(es, b, j)) {
                    if (k < q.cap) { q.pairs[2 * k] = b; q.pairs[2 * k + 1] = j; }
                    p.flag[j] = 1;
                    ++k;
                }
            }
            p.flag[b] = 1;
        }
    }
    if (b == 0) {
        p.st->nce_last = total;
        p.st->nce_total += total;
        p.st->steps_done += 1;
        if (total > q.cap) p.st->overflow = 1;
    }
    __syncthreads();                               // every pair test has read x1 before the jump moves it
    if (live) {
        p.x[b] = x + p.hj_over_mu * s0; p.x[ld + b] = y + p.hj_over_mu * s1; p.x[2 * ld + b] = z + p.hj_over_mu * s2;
    }
}

}  // namespace mopal
