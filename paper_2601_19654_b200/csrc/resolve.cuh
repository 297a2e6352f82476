// resolve.cuh - close-encounter resolution on the device (the paper's mdt_hkce, which it keeps on the
// host: PAPER.md:104 fn. 14, 126, 297-315; readings X-1..X-5 in DESIGN.md).
// The bodies of the encounter pair list are integrated as ONE system (X-1) from the snapshot x0, v0 over h
// under  dv/dt = -mu x/|x|^3 + sum over the listed pairs of gm_other (1 - K) (x_other - x)/r^3  (X-2) with
// Gragg's modified midpoint + Aitken-Neville extrapolation, n_k = 2, 4, .., 16 (X-3), step control by the
// accepting column only (X-4); every other body keeps its Kepler-drift result.
//
// First device version: one CTA, one thread per body of the system (<= RES_NMAX bodies, <= RES_PMAX pairs;
// more: the system is left to the drift and the failure is reported).  Per right-hand side: positions to shared
// memory, one thread per listed pair evaluates (1 - K)/r^3 (x_j - x_i) into shared memory, then every body sums
// its incident pairs in list order (its pairs as second member first - they precede its pairs as first member
// in the sorted list - X-5).  The extrapolation tableau of a body lives in its thread.
#pragma once
#include "common.cuh"
#include "encounters.cuh"

namespace mopal {

constexpr int RES_NMAX = 1024;     // bodies in the system = threads
constexpr int RES_PMAX = 2048;     // listed pairs
constexpr int RES_KMAX = 8;        // columns: 2, 4, .., 16 substeps
constexpr int RES_DYN_SMEM = RES_PMAX * 3 * 8;   // the pair terms of the current right-hand side (on top of 41 KB static)

struct ResStats { int bodies, steps, rhs, fail; };   // fail: 0 ok, 1 no convergence, 2 system too large

struct ResParams {
    const double *x0, *v0;       // snapshot (3*ld)
    double *x, *v;               // drifted state, in/out for the listed bodies
    const double *gm, *rcrit;
    const int* pairs;            // sorted (i, j) list of the last encounter pass
    const uint8_t* flag;         // 1 for every endpoint
    const DevStats* st;          // nce_last
    int* loc;                    // nb scratch: body -> index in the system
    double* tab;                 // 6 * RES_KMAX * RES_NMAX scratch: the extrapolation tableaux, [component][column][thread]
                                 // (kept out of local memory: a large per-thread stack makes the driver resize its
                                 // local-memory pool around every launch)
    ResStats* out;
    long long cap;
    int nb, ld;
    double mu, h, tol;
};

__device__ __forceinline__ double res_changeover(double s2, double rc) {     // A-1..A-5
    const double rc2 = rc * rc;
    if (s2 >= rc2) return 1.0;
    const double rin = 0.1 * rc;
    if (s2 <= rin * rin) return 0.0;
    const double q = (sqrt(s2) - rin) / (0.9 * rc);
    return q * q * q * (10.0 + q * (6.0 * q - 15.0));
}

__global__ void __launch_bounds__(RES_NMAX) resolve_kernel(ResParams p) {
    extern __shared__ __align__(16) unsigned char res_dyn[];
    __shared__ double sX[3 * RES_NMAX];                                 // positions of the current right-hand side
    __shared__ unsigned short sPi[RES_PMAX], sPj[RES_PMAX];             // local members of each listed pair
    __shared__ unsigned short sJadj[RES_PMAX];                          // pairs of each body as second member, list order
    __shared__ int sJstart[RES_NMAX + 1];
    __shared__ double sRed[32];
    __shared__ int sScan[64];
    double* sF = reinterpret_cast<double*>(res_dyn);                    // [RES_PMAX][3] pair terms

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const long long nce = p.st->nce_last;
    if (nce <= 0) { if (tid == 0) *p.out = ResStats{0, 0, 0, 0}; return; }
    if (nce > RES_PMAX || nce > p.cap) { if (tid == 0) *p.out = ResStats{0, 0, 0, 2}; return; }
    const int np = (int)nce;

    // ---- X-1: the system = flagged bodies in ascending order (thread t scans its own segment) ----
    const int seg = (p.nb + RES_NMAX - 1) / RES_NMAX;
    const int b0 = tid * seg, b1 = min(p.nb, b0 + seg);
    int cnt = 0;
    for (int b = b0; b < b1; ++b) cnt += p.flag[b] ? 1 : 0;
    if (tid < 64) sScan[tid] = 0;
    __syncthreads();
    int incl = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += t; }
    if (lane == 31) sScan[warp] = incl;
    __syncthreads();
    if (warp == 0) {
        int w = sScan[lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, w, o); if (lane >= o) w += t; }
        sScan[32 + lane] = w;
    }
    __syncthreads();
    const int n = sScan[63];
    if (n > RES_NMAX) { if (tid == 0) *p.out = ResStats{n, 0, 0, 2}; return; }
    {
        int k = (warp ? sScan[32 + warp - 1] : 0) + incl - cnt;
        for (int b = b0; b < b1; ++b)
            if (p.flag[b]) { p.loc[b] = k; sJstart[k] = b; ++k; }       // sJstart doubles as the body list for a moment
    }
    __syncthreads();
    const bool live = tid < n;
    const int me = live ? sJstart[tid] : 0;                            // my global body index
    __syncthreads();
    for (int q = tid; q < np; q += RES_NMAX) {
        sPi[q] = (unsigned short)p.loc[p.pairs[2 * q]];
        sPj[q] = (unsigned short)p.loc[p.pairs[2 * q + 1]];
    }
    __syncthreads();
    // adjacency: my pairs as first member are the contiguous range [iLo, iHi); my pairs as second member in list order
    int iLo = 0, iHi = 0, jCnt = 0;
    if (live) {
        int lo = 0, hi = np;
        while (lo < hi) { const int mid = (lo + hi) >> 1; if (sPi[mid] < tid) lo = mid + 1; else hi = mid; }
        iLo = lo; hi = np;
        while (lo < hi) { const int mid = (lo + hi) >> 1; if (sPi[mid] <= tid) lo = mid + 1; else hi = mid; }
        iHi = lo;
        for (int q = 0; q < iLo; ++q) jCnt += (sPj[q] == tid) ? 1 : 0;   // second member => first member smaller => q < iLo
    }
    {
        int inc2 = jCnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc2, o); if (lane >= o) inc2 += t; }
        if (lane == 31) sScan[warp] = inc2;
        __syncthreads();
        if (warp == 0) {
            int w = sScan[lane];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, w, o); if (lane >= o) w += t; }
            sScan[32 + lane] = w;
        }
        __syncthreads();
        const int off = (warp ? sScan[32 + warp - 1] : 0) + inc2 - jCnt;
        sJstart[tid] = off;
        if (tid == RES_NMAX - 1) sJstart[RES_NMAX] = off + jCnt;
        if (live) {
            int k = off;
            for (int q = 0; q < iLo; ++q) if (sPj[q] == tid) sJadj[k++] = (unsigned short)q;
        }
    }
    __syncthreads();
    const int jLo = sJstart[tid], jHi = jLo + jCnt;

    // ---- state and the right-hand side ----
    double y[6] = {0, 0, 0, 0, 0, 0};
    if (live) {
        for (int c = 0; c < 3; ++c) { y[c] = p.x0[(size_t)c * p.ld + me]; y[3 + c] = p.v0[(size_t)c * p.ld + me]; }
    }
    int nrhs = 0;
    auto rhs = [&](const double (&z)[6], double (&f)[6]) {
        __syncthreads();                                               // previous consumers of sX / sF are done
        if (live) { sX[tid] = z[0]; sX[RES_NMAX + tid] = z[1]; sX[2 * RES_NMAX + tid] = z[2]; }
        __syncthreads();
        for (int q = tid; q < np; q += RES_NMAX) {
            const int i = sPi[q], j = sPj[q];
            const double dx = sX[j] - sX[i], dy = sX[RES_NMAX + j] - sX[RES_NMAX + i], dz = sX[2 * RES_NMAX + j] - sX[2 * RES_NMAX + i];
            const double s2 = dx * dx + dy * dy + dz * dz;
            double u = 0.0;
            if (s2 > 0.0) {
                const double rc = fmax(p.rcrit[p.pairs[2 * q]], p.rcrit[p.pairs[2 * q + 1]]);
                u = (1.0 - res_changeover(s2, rc)) / (s2 * sqrt(s2));
            }
            sF[3 * q] = u * dx; sF[3 * q + 1] = u * dy; sF[3 * q + 2] = u * dz;
        }
        __syncthreads();
        if (live) {
            const double r2 = z[0] * z[0] + z[1] * z[1] + z[2] * z[2];
            const double w = -p.mu / (r2 * sqrt(r2));
            double a0 = w * z[0], a1 = w * z[1], a2 = w * z[2];
            for (int k = jLo; k < jHi; ++k) {                           // I am the second member: -gm_i u d
                const int q = sJadj[k];
                const double gi = p.gm[p.pairs[2 * q]];
                a0 -= gi * sF[3 * q]; a1 -= gi * sF[3 * q + 1]; a2 -= gi * sF[3 * q + 2];
            }
            for (int q = iLo; q < iHi; ++q) {                           // I am the first member: +gm_j u d
                const double gj = p.gm[p.pairs[2 * q + 1]];
                a0 += gj * sF[3 * q]; a1 += gj * sF[3 * q + 1]; a2 += gj * sF[3 * q + 2];
            }
            f[0] = z[3]; f[1] = z[4]; f[2] = z[5]; f[3] = a0; f[4] = a1; f[5] = a2;
        }
        ++nrhs;
    };

    const double hh = p.h;
    double t = 0.0, H = hh;
    int fail = 0, nacc = 0, halv = 0;
    double* T = p.tab + tid;                                           // T_{row, j} of component c at T[(c * RES_KMAX + j) * RES_NMAX]
    while (!fail) {
        const double rem = hh - t;
        if (fabs(rem) <= 4.0 * 2.220446049250313e-16 * fabs(hh)) break;
        bool last = false;
        if (fabs(H) >= fabs(rem)) { H = rem; last = true; }
        const double sx = sqrt(y[0] * y[0] + y[1] * y[1] + y[2] * y[2]);
        const double sv = sqrt(y[3] * y[3] + y[4] * y[4] + y[5] * y[5]);
        int acc = -1;
        for (int k = 0; k < RES_KMAX; ++k) {
            const int nsub = 2 * (k + 1);
            const double hs = H / (double)nsub;
            double z0[6], z1[6], f[6], res[6];
            rhs(y, f);
#pragma unroll
            for (int c = 0; c < 6; ++c) { z0[c] = y[c]; z1[c] = y[c] + hs * f[c]; }
            for (int m = 1; m < nsub; ++m) {
                rhs(z1, f);
#pragma unroll
                for (int c = 0; c < 6; ++c) { const double tt = z0[c] + 2.0 * hs * f[c]; z0[c] = z1[c]; z1[c] = tt; }
            }
            rhs(z1, f);
#pragma unroll
            for (int c = 0; c < 6; ++c) res[c] = 0.5 * (z0[c] + z1[c] + hs * f[c]);
            double err = 0.0;
#pragma unroll
            for (int c = 0; c < 6; ++c) {
                // row k of the tableau from row k-1 (in T), overwriting it column by column
                double* Tc = T + (size_t)c * RES_KMAX * RES_NMAX;
                double cur = res[c], prev = 0.0;
                for (int j = 1; j <= k; ++j) {
                    const double ratio = (double)(2 * (k + 1)) / (double)(2 * (k - j + 1));
                    const double old = Tc[(size_t)(j - 1) * RES_NMAX];
                    Tc[(size_t)(j - 1) * RES_NMAX] = cur;
                    prev = cur;
                    cur = cur + (cur - old) / (ratio * ratio - 1.0);
                }
                Tc[(size_t)k * RES_NMAX] = cur;
                if (k >= 1 && live) {
                    double e = fabs(cur - prev);
                    const double sc = c < 3 ? sx : sv;
                    e = sc > 0.0 ? e / sc : (e > 0.0 ? 1e300 : 0.0);
                    err = fmax(err, e);
                }
            }
            if (k >= 1) {                                               // block max of err
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) err = fmax(err, __shfl_xor_sync(0xffffffffu, err, o));
                __syncthreads();
                if (lane == 0) sRed[warp] = err;
                __syncthreads();
                double e = sRed[0];
                for (int w = 1; w < RES_NMAX / 32; ++w) e = fmax(e, sRed[w]);
                if (e <= p.tol) { acc = k; break; }
            }
        }
        if (acc < 0) {
            H *= 0.5;
            if (++halv > 40) fail = 1;
            continue;
        }
#pragma unroll
        for (int c = 0; c < 6; ++c) y[c] = T[((size_t)c * RES_KMAX + acc) * RES_NMAX];
        t = last ? hh : t + H;
        ++nacc;
        if (acc <= 3) H *= 2.0; else if (acc > 5) H *= 0.5;
    }
    if (!fail && live) {
        for (int c = 0; c < 3; ++c) { p.x[(size_t)c * p.ld + me] = y[c]; p.v[(size_t)c * p.ld + me] = y[3 + c]; }
    }
    if (tid == 0) *p.out = ResStats{n, nacc, nrhs, fail};
}

}  // namespace mopal
