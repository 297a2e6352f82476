// resolve.cuh - close-encounter resolution on the device (the paper's mdt_hkce, which it keeps on the
// host: PAPER.md:104 fn. 14, 126, 297-315; readings X-1..X-5 in DESIGN.md).
// The bodies of the encounter pair list are integrated (per component, X-1) from the snapshot x0, v0 over h
// under  dv/dt = -mu x/|x|^3 + sum over the listed pairs of gm_other (1 - K) (x_other - x)/r^3  (X-2) with
// Gragg's modified midpoint + Aitken-Neville extrapolation, n_k = 2, 4, .., 16 (X-3), step control by the
// accepting column only (X-4); every other body keeps its Kepler-drift result.
//
// The connected components of the pair graph are independent systems (X-1): resolve_label_kernel finds them,
// resolve_kernel gives each its own CTA, one thread per body (<= RES_NMAX bodies, <= RES_PMAX pairs per
// component; more: that component is left to the drift and counted as failed).  Per right-hand side: positions to shared
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
constexpr int RES_DYN_SMEM = RES_PMAX * (3 * 8 + 3 * 8 + 4);   // pair terms, per-pair gm_i, gm_j, rc, pair indices (+ 41 KB static)

struct ResStats { int bodies, steps, rhs, fail; };   // summed over the components; fail = components not resolved

struct ResParams {
    const double *x0, *v0;       // snapshot (3*ld)
    double *x, *v;               // drifted state, in/out for the listed bodies
    const double *gm, *rcrit;
    const int* pairs;            // sorted (i, j) list of the last encounter pass
    const uint8_t* flag;         // 1 for every endpoint
    DevStats* st;                // nce_last; resolve_fail (cumulative)
    int* loc;                    // nb scratch: body -> index in its component
    int* label;                  // nb scratch: smallest body of the component (valid for flagged bodies)
    int* roots; int* nroots;     // the components' smallest bodies
    int* done;                   // per component: 1 once an instance of resolve_kernel has taken it
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

// exclusive block scan of one int per thread (blocks of up to 1024 threads); sScan: 64 ints, the slots of
// warps the block does not have stay 0
__device__ __forceinline__ int res_scan(int v, int* sScan, int& total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += t; }
    __syncthreads();                                   // previous users of sScan are done
    if (lane == 31) sScan[warp] = incl;
    __syncthreads();
    if (warp == 0) {
        int w = sScan[lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, w, o); if (lane >= o) w += t; }
        sScan[32 + lane] = w;
    }
    __syncthreads();
    total = sScan[63];
    return (warp ? sScan[32 + warp - 1] : 0) + incl - v;
}

// X-1: connected components of the pair graph.  One CTA: label[b] = smallest body of b's component, by
// min-propagation along the listed pairs until nothing changes (encounter graphs are stars around the
// big bodies: a few sweeps), then the list of roots (a root is the first member of its first pair).
__global__ void __launch_bounds__(RES_NMAX) resolve_label_kernel(ResParams p) {
    const int tid = threadIdx.x;
    if (tid == 0) { *p.out = ResStats{0, 0, 0, 0}; *p.nroots = 0; }
    const long long nce = p.st->nce_last;
    if (nce <= 0) return;
    if (nce > p.cap) { if (tid == 0) { p.out->fail = 1 << 30; atomicAdd(&p.st->resolve_fail, 1); } return; }      // truncated list: nothing can be resolved
    const int np = (int)nce;
    volatile int* label = p.label;
    for (int q = tid; q < np; q += RES_NMAX) { label[p.pairs[2 * q]] = p.pairs[2 * q]; label[p.pairs[2 * q + 1]] = p.pairs[2 * q + 1]; }
    __syncthreads();
    int changed;
    do {
        changed = 0;
        for (int q = tid; q < np; q += RES_NMAX) {
            const int i = p.pairs[2 * q], j = p.pairs[2 * q + 1];
            const int li = label[i], lj = label[j];
            if (li < lj) { atomicMin(p.label + j, li); changed = 1; }
            else if (lj < li) { atomicMin(p.label + i, lj); changed = 1; }
        }
        changed = __syncthreads_or(changed);
    } while (changed);
    for (int q = tid; q < np; q += RES_NMAX) {
        const int i = p.pairs[2 * q];
        if (label[i] == i && (q == 0 || p.pairs[2 * (q - 1)] != i)) { const int c = atomicAdd(p.nroots, 1); p.roots[c] = i; p.done[c] = 0; }
    }
}

// One CTA per component (CTAs walk the root list), one thread per body of the component.  Three instances by
// the component's number of pairs, PLO < np <= PHI, with NT = 2 PHI threads (a component of np pairs has at
// most 2 np bodies; the last instance takes what fits 1024 bodies): most components are single pairs, and the
// barriers of every right-hand side cost by the warp - 64 threads for np <= 32, 256 for np <= 128, then 512
// threads if the bodies fit (the stars around the big bodies), else 1024.
// LAST: the instance that takes whatever the earlier ones left (they skip a component whose bodies outnumber
// their threads; the last one counts it as failed).
template <int NT, int PLO, int PHI, bool LAST>
__global__ void __launch_bounds__(NT) resolve_kernel(ResParams p) {
    extern __shared__ __align__(16) unsigned char res_dyn[];
    __shared__ double sX[3 * NT];                                 // positions of the current right-hand side
    __shared__ unsigned short sPi[RES_PMAX], sPj[RES_PMAX];             // local members of each pair of the component
    __shared__ unsigned short sJadj[RES_PMAX];                          // pairs of each body as second member, list order
    __shared__ int sJstart[NT + 1];
    __shared__ double sRed[32];
    __shared__ int sScan[64];
    __shared__ int sHub[6];                                             // the body with most pairs: thread, jLo, jCnt, iLo, iHi, degree
    __shared__ double sHubAcc[3];
    double* sF = reinterpret_cast<double*>(res_dyn);                    // [RES_PMAX][3] pair terms
    double* sGi = sF + 3 * RES_PMAX;                                    // [RES_PMAX] gm of the first member
    double* sGj = sGi + RES_PMAX;                                       // [RES_PMAX] gm of the second member
    double* sRc = sGj + RES_PMAX;                                       // [RES_PMAX] max(rcrit_i, rcrit_j)
    int* sPq = reinterpret_cast<int*>(sRc + RES_PMAX);                  // [RES_PMAX] index of the pair in the list

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid < 64) sScan[tid] = 0;
    __syncthreads();
    const int ncomp = *p.nroots;
    const int npAll = (int)p.st->nce_last;
    for (int comp = blockIdx.x; comp < ncomp; comp += gridDim.x) {
    const int root = p.roots[comp];
    __syncthreads();                                                   // the previous component is finished with shared memory

    // ---- the component's pairs, in list order ----
    int np = 0;
    for (int base = 0; base < npAll; base += NT) {
        const int q = base + tid;
        const int mine = (q < npAll && p.label[p.pairs[2 * q]] == root) ? 1 : 0;
        int tot;
        const int off = res_scan(mine, sScan, tot);
        if (mine && np + off < RES_PMAX) sPq[np + off] = q;
        np += tot;
    }
    if (np <= PLO || np > PHI || p.done[comp]) continue;               // another instance's component
    if (np > RES_PMAX) { if (LAST && tid == 0) { atomicAdd(&p.out->fail, 1); atomicAdd(&p.st->resolve_fail, 1); } continue; }
    // ---- its bodies in ascending order (thread t scans its own segment of the flags) ----
    // (segments of a multiple of 8 bodies: the flags are read eight at a time where the array is 8-byte aligned -
    // at 1e6 bodies almost all of them are 0)
    const int seg = ((p.nb + NT - 1) / NT + 7) & ~7;
    const int b0 = min(p.nb, tid * seg), b1 = min(p.nb, b0 + seg);
    const bool wide = (reinterpret_cast<uintptr_t>(p.flag) & 7u) == 0;
    int cnt = 0;
    for (int b = b0; b < b1; b += 8) {
        if (wide && b + 8 <= b1 && *reinterpret_cast<const unsigned long long*>(p.flag + b) == 0ull) continue;
        const int e = min(b + 8, b1);
        for (int q = b; q < e; ++q) cnt += (p.flag[q] && p.label[q] == root) ? 1 : 0;
    }
    int n;
    {
        int k = res_scan(cnt, sScan, n);
        if (n <= NT && cnt > 0)
            for (int b = b0; b < b1; ++b)
                if (p.flag[b] && p.label[b] == root) { p.loc[b] = k; sJstart[k] = b; ++k; }   // sJstart doubles as the body list
    }
    if (n > NT) {
        if (LAST && tid == 0) { atomicAdd(&p.out->fail, 1); atomicAdd(&p.st->resolve_fail, 1); atomicAdd(&p.out->bodies, n); }
        continue;                                                      // not LAST: a later, wider instance takes it
    }
    if (tid == 0) p.done[comp] = 1;
    __syncthreads();
    const bool live = tid < n;
    const int me = live ? sJstart[tid] : 0;                            // my global body index
    __syncthreads();
    for (int q = tid; q < np; q += NT) {
        const int bi = p.pairs[2 * sPq[q]], bj = p.pairs[2 * sPq[q] + 1];
        sPi[q] = (unsigned short)p.loc[bi];
        sPj[q] = (unsigned short)p.loc[bj];
        sGi[q] = p.gm[bi]; sGj[q] = p.gm[bj];
        sRc[q] = fmax(p.rcrit[bi], p.rcrit[bj]);
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
    int jLo;
    {
        int tot;
        jLo = res_scan(jCnt, sScan, tot);
        if (live) {
            int k = jLo;
            for (int q = 0; q < iLo; ++q) if (sPj[q] == tid) sJadj[k++] = (unsigned short)q;
        }
    }
    __syncthreads();
    const int jHi = jLo + jCnt;
    // the component's hub (a giant with hundreds of pairs): its sum is taken by warp 0 together, lane l adding the
    // terms l, l + 32, .. and a fixed shuffle tree - every other body sums its few terms alone
    {
        const int deg = live ? jCnt + (iHi - iLo) : 0;
        int best = (deg << 11) | (NT - 1 - tid);                        // max degree, ties to the smallest thread
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) best = max(best, __shfl_xor_sync(0xffffffffu, best, o));
        __syncthreads();
        if (lane == 0) sScan[warp] = best;
        __syncthreads();
        int bb = sScan[0];
        for (int w = 1; w < NT / 32; ++w) bb = max(bb, sScan[w]);
        __syncthreads();
        if (tid < 64) sScan[tid] = 0;                                   // the scan helper expects zeros in unused slots
        const int hubTid = NT - 1 - (bb & 2047);
        if (tid == hubTid) { sHub[0] = tid; sHub[1] = jLo; sHub[2] = jCnt; sHub[3] = iLo; sHub[4] = iHi; sHub[5] = deg; }
        __syncthreads();
    }
    const bool hubOn = sHub[5] > 64;                                    // CTA-uniform
    const bool iAmHub = hubOn && tid == sHub[0];

    // ---- state and the right-hand side ----
    double y[6] = {0, 0, 0, 0, 0, 0};
    if (live) {
        for (int c = 0; c < 3; ++c) { y[c] = p.x0[(size_t)c * p.ld + me]; y[3 + c] = p.v0[(size_t)c * p.ld + me]; }
    }
    int nrhs = 0;
    auto rhs = [&](const double (&z)[6], double (&f)[6]) {
        __syncthreads();                                               // previous consumers of sX / sF are done
        if (live) { sX[tid] = z[0]; sX[NT + tid] = z[1]; sX[2 * NT + tid] = z[2]; }
        __syncthreads();
        for (int q = tid; q < np; q += NT) {
            const int i = sPi[q], j = sPj[q];
            const double dx = sX[j] - sX[i], dy = sX[NT + j] - sX[NT + i], dz = sX[2 * NT + j] - sX[2 * NT + i];
            const double s2 = dx * dx + dy * dy + dz * dz;
            double u = 0.0;
            if (s2 > 0.0) {
                u = (1.0 - res_changeover(s2, sRc[q])) / (s2 * sqrt(s2));
            }
            sF[3 * q] = u * dx; sF[3 * q + 1] = u * dy; sF[3 * q + 2] = u * dz;
        }
        __syncthreads();
        if (hubOn) {
            if (warp == 0) {
                const int hj0 = sHub[1], hjc = sHub[2], hi0 = sHub[3], D = sHub[5];
                double h0 = 0.0, h1 = 0.0, h2 = 0.0;
                for (int t = lane; t < D; t += 32) {
                    if (t < hjc) { const int q = sJadj[hj0 + t]; const double gi = sGi[q]; h0 -= gi * sF[3 * q]; h1 -= gi * sF[3 * q + 1]; h2 -= gi * sF[3 * q + 2]; }
                    else { const int q = hi0 + (t - hjc); const double gj = sGj[q]; h0 += gj * sF[3 * q]; h1 += gj * sF[3 * q + 1]; h2 += gj * sF[3 * q + 2]; }
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    h0 += __shfl_xor_sync(0xffffffffu, h0, o); h1 += __shfl_xor_sync(0xffffffffu, h1, o); h2 += __shfl_xor_sync(0xffffffffu, h2, o);
                }
                if (lane == 0) { sHubAcc[0] = h0; sHubAcc[1] = h1; sHubAcc[2] = h2; }
            }
            __syncthreads();
        }
        if (live) {
            const double r2 = z[0] * z[0] + z[1] * z[1] + z[2] * z[2];
            const double w = -p.mu / (r2 * sqrt(r2));
            double a0 = w * z[0], a1 = w * z[1], a2 = w * z[2];
            if (iAmHub) { a0 += sHubAcc[0]; a1 += sHubAcc[1]; a2 += sHubAcc[2]; }
            else {
            for (int k = jLo; k < jHi; ++k) {                           // I am the second member: -gm_i u d
                const int q = sJadj[k];
                const double gi = sGi[q];
                a0 -= gi * sF[3 * q]; a1 -= gi * sF[3 * q + 1]; a2 -= gi * sF[3 * q + 2];
            }
            for (int q = iLo; q < iHi; ++q) {                           // I am the first member: +gm_j u d
                const double gj = sGj[q];
                a0 += gj * sF[3 * q]; a1 += gj * sF[3 * q + 1]; a2 += gj * sF[3 * q + 2];
            }
            }
            f[0] = z[3]; f[1] = z[4]; f[2] = z[5]; f[3] = a0; f[4] = a1; f[5] = a2;
        }
        ++nrhs;
    };

    const double hh = p.h;
    double t = 0.0, H = hh;
    int fail = 0, nacc = 0, halv = 0;
    // the tableaux: shared memory for the instances of up to 256 threads, global scratch above
    double* T = (NT <= 256 ? reinterpret_cast<double*>(res_dyn + RES_DYN_SMEM) : p.tab + (size_t)blockIdx.x * 6 * RES_KMAX * NT) + tid;                                           // T_{row, j} of component c at T[(c * RES_KMAX + j) * threads]
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
                // row k of the tableau from row k-1 (in T), overwriting it column by column; the old row is read
                // first, all loads in flight together (interleaved with the stores they would serialise)
                double* Tc = T + (size_t)c * RES_KMAX * NT;
                double old[RES_KMAX];
#pragma unroll
                for (int j = 0; j < RES_KMAX; ++j) old[j] = (j < k) ? Tc[(size_t)j * NT] : 0.0;
                double cur = res[c], prev = 0.0;
#pragma unroll
                for (int j = 1; j < RES_KMAX; ++j) {
                    if (j <= k) {
                        const double ratio = (double)(2 * (k + 1)) / (double)(2 * (k - j + 1));
                        Tc[(size_t)(j - 1) * NT] = cur;
                        prev = cur;
                        cur = cur + (cur - old[j - 1]) / (ratio * ratio - 1.0);
                    }
                }
                Tc[(size_t)k * NT] = cur;
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
                for (int w = 1; w < NT / 32; ++w) e = fmax(e, sRed[w]);
                if (e <= p.tol) { acc = k; break; }
            }
        }
        if (acc < 0) {
            H *= 0.5;
            if (++halv > 40) fail = 1;
            continue;
        }
#pragma unroll
        for (int c = 0; c < 6; ++c) y[c] = T[((size_t)c * RES_KMAX + acc) * NT];
        t = last ? hh : t + H;
        ++nacc;
        halv = 0;                                                       // X-4: 40 halvings in a row are a failure
        if (acc <= 3) H *= 2.0; else if (acc > 5) H *= 0.5;
    }
    if (!fail && live) {
        for (int c = 0; c < 3; ++c) { p.x[(size_t)c * p.ld + me] = y[c]; p.v[(size_t)c * p.ld + me] = y[3 + c]; }
    }
    if (tid == 0) {
        atomicAdd(&p.out->bodies, n); atomicAdd(&p.out->steps, nacc); atomicAdd(&p.out->rhs, nrhs);
        if (fail) { atomicAdd(&p.out->fail, 1); atomicAdd(&p.st->resolve_fail, 1); }
    }
    }   // components
}

}  // namespace mopal
