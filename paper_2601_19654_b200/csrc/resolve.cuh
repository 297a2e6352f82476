// resolve.cuh - close-encounter resolution on the device (the paper's mdt_hkce, which it keeps on the
// host: PAPER.md:104 fn. 14, 126, 297-315; readings X-1..X-3, X-5 in DESIGN.md).
// The bodies of the encounter pair list are integrated (per connected component of the pair graph, X-1) from
// the snapshot x0, v0 over h under
//     dv/dt = -mu x/|x|^3 + sum over the listed pairs of gm_other (1 - K) (x_other - x)/r^3        (X-2)
// with Gragg's modified midpoint + Aitken-Neville extrapolation, n_k = 2, 4, .., 16 (X-3); every other body
// keeps its Kepler-drift result.  The step-size / order control is the kernel's own (Hairer-Wanner style work-per-
// unit-step controller, section "controller" below) - the oracle keeps its simple rule X-4; the two agree to the
// tolerance, not step for step.
//
// Kernels:
//   resolve_label_kernel   one CTA: connected components by min-label propagation over the pair list, components
//                          numbered in ascending order of their smallest body, their pairs grouped (cq), and one
//                          work list per size class.
//   resolve_solve_kernel<NT, CLS>   one CTA per component, taken from the class list by ticket, one thread per body.
//                          Classes 0..3: np <= 63 / 255 / 511 / 1023 pairs with 64 / 256 / 512 / 1024 threads.
//                          Everything a right-hand side touches is in shared memory, carved by the component's
//                          actual size; the extrapolation tableau too when it fits (else global scratch).
//   resolve_small_kernel   class 5, at most 31 pairs (almost every system): one CTA of 8 warps, warp w = column w of the
//                          Bulirsch-Stoer step, lane = body / pair.
//   resolve_stream_kernel  class 4, any size: the same algorithm with all per-body and per-pair state in global
//                          pools, thread-strided loops, block-wide sums for the hubs.
//
// A right-hand side costs two block barriers: positions -> shared memory | one thread per listed pair evaluates
// (1 - K)/r^3 (x_j - x_i) into shared memory | every body sums its incident terms in list order (its pairs as
// second member first, X-5); a body with more than RES_HEAVY pairs (a giant: the hub of a star of hundreds) is
// summed by its warp together, lane l taking the terms l, l + 32, .. and a fixed shuffle tree - deterministic.
// The midpoint rule runs on INCREMENTS (d = z - y): the error estimate |T_kk - T_k,k-1| is then formed from numbers of
// the size of the step's change, not of the state, so its rounding floor sits far below any sensible tolerance, and
// f(y) is evaluated once per Bulirsch-Stoer step instead of once per column.
#pragma once
#include "common.cuh"
#include "encounters.cuh"

namespace mopal {

constexpr int RES_KMAX = 8;        // columns: 2, 4, .., 16 substeps
constexpr int RES_HEAVY = 12;      // a body with more pairs is summed by its whole warp
constexpr int RES_NCLS = 10;       // size classes: 0..3 one thread per body (64 / 256 / 512 / 1024 threads), 4 streamed,
                                   // 5 the small systems (at most RES_PHI_S pairs): one warp per column; 6 those of
                                   // them that look like a long chain of steps (a deep passage), in four levels of
                                   // depth (6: the deepest .. 9): taken first, deepest first
constexpr int RES_PHI_0 = 63, RES_PHI_1 = 255, RES_PHI_2 = 511, RES_PHI_3 = 1023;   // largest pair count of classes 0..3
constexpr int RES_PHI_S = 31;      // ... and of class 5: at most 32 bodies, one per lane
constexpr int RES_S_THREADS = 32 * RES_KMAX;   // resolve_small_kernel: warp w integrates column w
constexpr int RES_CTL_CNT = 1, RES_CTL_TKT = 1 + RES_NCLS, RES_CTL_POOL = 1 + 2 * RES_NCLS, RES_CTL_N = 2 + 2 * RES_NCLS;
constexpr int RES_LABEL_THREADS = 1024;
constexpr int RES_NCOL = 8;        // CTAs per cluster = columns side by side (classes 1..3)
constexpr int RES_NCLUSTERS = 24;  // clusters of the three launches together (8 + 8 + 8)
constexpr int RES_D_THREADS = 1024;
constexpr int RES_D_BODY_PLANES = 3 + 6 + 6 + 6 + 3 + 2 + 3 + 6 * RES_KMAX;   // P, Y, D0, D1, F0A, SC, ACC, T
constexpr int RES_D_BODY_IPLANES = 7;                                    // body, iLo, iHi, jLo, d2, tier, list of the warp-summed bodies
constexpr int RES_D_PAIR_PLANES = 10;                                    // F(3), rc2, inv, gi, gj, Dy(3)
constexpr int RES_D_PAIR_IPLANES = 7;                                    // q, global i, global j, local i, local j, adjacency (sorted, unsorted)
constexpr int RES_D_HMAX = 32;     // hubs of one class-D component summed by the whole block

struct ResStats { int bodies, steps, rhs, fail; };   // summed over the components; fail = components not resolved

struct ResParams {
    const double *x0, *v0;       // snapshot (3*ld)
    double *x, *v;               // drifted state, in/out for the listed bodies
    const double *gm, *rcrit;
    const int* pairs;            // sorted (i, j) list of the last encounter pass
    DevStats* st;                // nce_last; resolve_fail (cumulative)
    ResStats* out;
    int* loc;                    // nb: label kernel: root body -> component; solve kernels: body -> index in its component
    int* label;                  // nb: smallest body of the component (valid for listed bodies)
    int* aux;                    // nb: the component a body is in (-1: none; a detached body, or a massive body with detached partners only)
    int* cown;                   // per system: the detached body it belongs to (the only one written back), or -1
    int* ckey;                   // per system: smallest (closest straight-line approach / rc)^2 of its own pairs, as float bits
    int *cnp, *cstart, *cfill;   // per system (<= cap): pairs (a detached body's: with its partners' components), first slot in cq, own pairs there
    int* cq;                     // cap: pair indices grouped by component (unordered inside a group)
    int* clist;                  // RES_NCLS * cap: the components of each class
    int* ctl;                    // [0] components, [RES_CTL_CNT + c] class counts, [RES_CTL_TKT + c] tickets, [RES_CTL_POOL] streamed-class body pool in use
    int* mode;                   // [1] <- 1 if this list holds a component of more than 63 pairs (a long chain: mopal.cu), else 0
    double* tab;                 // extrapolation tableaux of the class-C CTAs whose component does not leave room in shared memory
    double* dbody; int* dbodyi;  // class D pools: planes of dbodyN doubles / ints
    double* dpair; int* dpairi;  // planes of cap
    long long dbodyN;
    long long cap;
    int nb, ld;
    double mu, h, tol;
};

// 1 / ((n_k / n_{k-j})^2 - 1), n_k = 2 (k + 1): Aitken-Neville weights of the (H/n)^2 extrapolation
__constant__ double RES_COEF[RES_KMAX * RES_KMAX] = {
    0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0,
    0.0, 1.0 / 3.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0,
    0.0, 4.0 / 5.0, 1.0 / 8.0, 0.0, 0.0, 0.0, 0.0, 0.0,
    0.0, 9.0 / 7.0, 4.0 / 12.0, 1.0 / 15.0, 0.0, 0.0, 0.0, 0.0,
    0.0, 16.0 / 9.0, 9.0 / 16.0, 4.0 / 21.0, 1.0 / 24.0, 0.0, 0.0, 0.0,
    0.0, 25.0 / 11.0, 16.0 / 20.0, 9.0 / 27.0, 4.0 / 32.0, 1.0 / 35.0, 0.0, 0.0,
    0.0, 36.0 / 13.0, 25.0 / 24.0, 16.0 / 33.0, 9.0 / 40.0, 4.0 / 45.0, 1.0 / 48.0, 0.0,
    0.0, 49.0 / 15.0, 36.0 / 28.0, 25.0 / 39.0, 16.0 / 48.0, 9.0 / 55.0, 4.0 / 60.0, 1.0 / 63.0,
};

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

__device__ __forceinline__ int res_class(int np) { return np <= RES_PHI_S ? 5 : np <= RES_PHI_0 ? 0 : np <= RES_PHI_1 ? 1 : np <= RES_PHI_2 ? 2 : np <= RES_PHI_3 ? 3 : 4; }

__device__ __forceinline__ void res_bar(int nthreads);

// producer / consumer halves of named barrier id (n threads in all): the producers arrive and go on, the consumers wait
__device__ __forceinline__ void res_nb_arrive(int id, int n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void res_nb_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }

// thread-block cluster: the hardware barrier in its two halves, and a load from another CTA's shared memory
__device__ __forceinline__ void res_cl_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void res_cl_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }
__device__ __forceinline__ void res_cl_sync() { res_cl_arrive(); res_cl_wait(); }
__device__ __forceinline__ double res_ld_remote(const void* mine, int rank) {      // the same variable in CTA `rank` of the cluster
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(smem_u32(mine)), "r"(rank));
    double v;
    asm volatile("ld.shared::cluster.f64 %0, [%1];" : "=d"(v) : "r"(r) : "memory");
    return v;
}

// barrier of the first nthreads threads of the block (whole warps), beside the block barrier 0
__device__ __forceinline__ void res_bar(int nthreads) { asm volatile("bar.sync 1, %0;" ::"r"(nthreads) : "memory"); }

// The system a listed pair belongs to ("owner" body).  A massless body exerts no force: a pair of two massless bodies
// carries no term at all (it is left out), and a massless body can be DETACHED - integrated in a system of its own:
// itself, its massive partners and the components ("cores") those partners belong to, none of which feels it (they are
// integrated along, not written back) - instead of chaining thousands of test particles and their giant into one
// system with one step size.  The solutions are the same: nothing a detached body does reaches another body.  A
// massless body is detached when its system stays small (at most RES_DET_PARTNERS massive partners, at most RES_PHI_0
// pairs with the cores counted in); otherwise it is an ordinary member of its partners' component.
// label of a massless body: -1 detached, else (its own index to start with) the component's smallest body.
constexpr int RES_DET_PARTNERS = 8;
__device__ __forceinline__ int res_owner(const ResParams& p, int q, const int* label) {
    const int i = p.pairs[2 * q], j = p.pairs[2 * q + 1];
    const bool mi = p.gm[i] > 0.0, mj = p.gm[j] > 0.0;
    if (!mi && !mj) return -1;                                   // no force either way
    if (!mi && label[i] < 0) return i;                           // i detached
    if (!mj && label[j] < 0) return j;                           // j detached
    return label[i];                                             // the component's smallest body
}

// How deep a listed pair's passage looks (scheduling only: the systems that will need many Bulirsch-Stoer steps are started
// first, so that the longest chain of the list runs beside the others instead of after them): the closest approach of the
// straight line from the separation at the snapshot to the separation after the drift, squared, over rc^2 - as the bits
// of a non-negative float, which order like the floats.
constexpr float RES_DEEP_RATIO = 0.04f;           // closest approach below 0.2 rc
__device__ __forceinline__ int res_depth_key(const ResParams& p, int q) {
    const int i = p.pairs[2 * q], j = p.pairs[2 * q + 1];
    float a[3], d[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        a[c] = (float)(p.x0[(size_t)c * p.ld + j] - p.x0[(size_t)c * p.ld + i]);
        d[c] = (float)(p.x[(size_t)c * p.ld + j] - p.x[(size_t)c * p.ld + i]) - a[c];
    }
    const float dd = d[0] * d[0] + d[1] * d[1] + d[2] * d[2], ad = a[0] * d[0] + a[1] * d[1] + a[2] * d[2];
    const float t = dd > 0.f ? fminf(fmaxf(-ad / dd, 0.f), 1.f) : 0.f;
    const float m0 = a[0] + t * d[0], m1 = a[1] + t * d[1], m2 = a[2] + t * d[2];
    const float rc = (float)fmax(p.rcrit[i], p.rcrit[j]);
    const float r = rc > 0.f ? (m0 * m0 + m1 * m1 + m2 * m2) / (rc * rc) : 1e30f;
    return __float_as_int(r >= 0.f ? fminf(r, 1e30f) : 1e30f);            // NaN: not deep
}

// X-1: connected components of the pair graph and the detached bodies' systems.  One cluster of RES_LABEL_CTAS CTAs (a list
// of up to RES_LABEL_SOLO pairs: its first CTA alone): label[b] = smallest body of b's component, by min-propagation along
// the pairs until nothing changes (encounter graphs are stars around the big bodies: a few sweeps); then the systems in
// ascending order of their first pair, their pair counts, the pairs grouped by system and the class lists.  Every phase
// is a loop over the pairs (or the systems) strided over all the threads at work, with the cluster's hardware barrier
// in between; the two exchanges that are not through global memory - "did any thread change a label" and the CTAs' totals
// of a scan - go through the CTAs' shared memory.  (One CTA took 0.37 ms for the 12.7 k pairs of the big x all workload.)
constexpr int RES_LABEL_CTAS = 8;
constexpr int RES_LABEL_SOLO = 2048;
__device__ __forceinline__ int res_ld_remote_int(const void* mine, int rank) {    // the same variable in CTA `rank` of the cluster
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(smem_u32(mine)), "r"(rank));
    int v;
    asm volatile("ld.shared::cluster.s32 %0, [%1];" : "=r"(v) : "r"(r) : "memory");
    return v;
}
__global__ void __launch_bounds__(RES_LABEL_THREADS) resolve_label_kernel(ResParams p) {
    __shared__ int sScan[64];
    __shared__ int sXc[2][2];                                              // [parity][flag | total]: what this CTA tells the others
    constexpr int NT = RES_LABEL_THREADS;
    const int tid = threadIdx.x, rank = blockIdx.x;                        // (the grid is one cluster)
    if (tid < 64) sScan[tid] = 0;
    const long long nce = p.st->nce_last;
    // a short list is one CTA's work (its barriers are cheaper than the cluster's); the other CTAs leave at once and the
    // cluster's barrier is never used
    const bool solo = nce <= RES_LABEL_SOLO || gridDim.x == 1;
    if (solo && rank > 0) return;
    const int NC = solo ? 1 : (int)gridDim.x;
    const int gtid = rank * NT + tid, GNT = NC * NT;
    if (gtid == 0) { *p.out = ResStats{0, 0, 0, 0}; for (int k = 0; k < RES_CTL_N; ++k) p.ctl[k] = 0; }
    if (nce <= 0 || nce > p.cap) { if (gtid == 0) p.mode[1] = 0; }
    if (nce <= 0) return;
    if (nce > p.cap) { if (gtid == 0) { p.out->fail = 1 << 30; atomicAdd(&p.st->resolve_fail, 1); } return; }      // truncated list: nothing can be resolved
    int xph = 0;                                                           // exchanges so far (the slots alternate)
    // barrier of all the threads at work; what a thread wrote to global memory before it, every thread sees after it
    auto sync = [&]() { if (solo) __syncthreads(); else res_cl_sync(); };
    // OR over all the threads at work (with a barrier)
    auto any = [&](int v) -> int {
        v = __syncthreads_or(v);
        if (solo) return v;
        if (tid == 0) sXc[xph & 1][0] = v;
        res_cl_sync();
        int r = 0;
        for (int c = 0; c < NC; ++c) r |= res_ld_remote_int(&sXc[xph & 1][0], c);
        ++xph;
        return r;
    };
    // exclusive scan of one int per thread, in (CTA, thread) order, and the total over all the threads at work
    auto scan = [&](int v, int& total) -> int {
        int tot;
        const int off = res_scan(v, sScan, tot);
        if (solo) { total = tot; return off; }
        if (tid == 0) sXc[xph & 1][1] = tot;
        res_cl_sync();
        int before = 0, all = 0;
        for (int c = 0; c < NC; ++c) { const int t = res_ld_remote_int(&sXc[xph & 1][1], c); all += t; before += c < rank ? t : 0; }
        ++xph;
        total = all;
        return before + off;
    };
    // min-label propagation along the pairs that belong to components (not left out, not owned by a detached body)
    auto propagate = [&](bool massive_only) {
        volatile int* label = p.label;
        int changed;
        do {
            changed = 0;
            for (int q = gtid; q < (int)nce; q += GNT) {
                const int i = p.pairs[2 * q], j = p.pairs[2 * q + 1];
                const bool mi = p.gm[i] > 0.0, mj = p.gm[j] > 0.0;
                if (massive_only ? !(mi && mj) : (!mi && !mj)) continue;
                const int li = label[i], lj = label[j];
                if (li < 0 || lj < 0) continue;                   // a detached body's pair
                if (li < lj) { atomicMin(p.label + j, li); changed = 1; }
                else if (lj < li) { atomicMin(p.label + i, lj); changed = 1; }
            }
            changed = any(changed);
        } while (changed);
    };
    const int np = (int)nce;
    int anyMassless = 0;
    for (int q = gtid; q < np; q += GNT) {
        const int i = p.pairs[2 * q], j = p.pairs[2 * q + 1];
        p.label[i] = i; p.label[j] = j; p.aux[i] = 0; p.aux[j] = 0; p.loc[i] = 0; p.loc[j] = 0;
        anyMassless |= (p.gm[i] > 0.0 && p.gm[j] > 0.0) ? 0 : 1;
    }
    anyMassless = any(anyMassless);
    if (anyMassless) {
        // cores: components of the massive-massive pairs alone; aux[root] = their pair count
        propagate(true);
        for (int q = gtid; q < np; q += GNT) {
            const int i = p.pairs[2 * q], j = p.pairs[2 * q + 1];
            if (p.gm[i] > 0.0 && p.gm[j] > 0.0) atomicAdd(&p.aux[p.label[i]], 1);
        }
        sync();
        // size of a massless body's own system (an upper bound: a core shared by two partners counts twice)
        for (int q = gtid; q < np; q += GNT) {
            const int i = p.pairs[2 * q], j = p.pairs[2 * q + 1];
            const bool mi = p.gm[i] > 0.0, mj = p.gm[j] > 0.0;
            if (mi == mj) continue;
            const int l = mi ? j : i, h = mi ? i : j;
            atomicAdd(&p.loc[l], 1);                                              // partners
            atomicAdd(&p.aux[l], 1 + p.aux[p.label[h]]);                           // pairs (aux of a massless body)
        }
        sync();
        for (int q = gtid; q < np; q += GNT) {
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int b = p.pairs[2 * q + e];
                if (!(p.gm[b] > 0.0)) p.label[b] = (p.loc[b] >= 1 && p.loc[b] <= RES_DET_PARTNERS && p.aux[b] <= RES_PHI_0) ? -1 : b;
            }
        }
        sync();
    }
    propagate(false);
    // first pair of every owner (loc, until the systems are numbered)
    for (int q = gtid; q < np; q += GNT) { p.loc[p.pairs[2 * q]] = 0x7fffffff; p.loc[p.pairs[2 * q + 1]] = 0x7fffffff; }
    sync();
    for (int q = gtid; q < np; q += GNT) {
        const int o = res_owner(p, q, p.label);
        if (o >= 0) atomicMin(&p.loc[o], q);
    }
    sync();
    int carry = 0;
    for (int base = 0; base < np; base += GNT) {
        const int q = base + gtid;
        int isfirst = 0, o = -1;
        if (q < np) { o = res_owner(p, q, p.label); isfirst = (o >= 0 && p.loc[o] == q) ? 1 : 0; }
        int tot;
        const int off = scan(isfirst, tot);
        if (isfirst) { const int c = carry + off; p.cfill[c] = q; p.cnp[c] = 0; p.cown[c] = p.gm[o] > 0.0 ? -1 : o; p.ckey[c] = 0x7f7fffff; }
        carry += tot;
    }
    const int ncomp = carry;
    sync();
    for (int c = gtid; c < ncomp; c += GNT) { p.loc[res_owner(p, p.cfill[c], p.label)] = c; }   // owner -> system
    sync();
    // aux[b] = the component of a body that is in one (massive, or massless and not detached), else -1
    for (int q = gtid; q < np; q += GNT) {
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const int b = p.pairs[2 * q + e];
            const int lb = p.label[b];
            p.aux[b] = (lb >= 0 && p.loc[lb] != 0x7fffffff) ? p.loc[lb] : -1;
        }
    }
    for (int c = gtid; c < ncomp; c += GNT) p.cfill[c] = 0;
    sync();
    for (int q = gtid; q < np; q += GNT) {
        const int o = res_owner(p, q, p.label);
        if (o >= 0) { atomicAdd(&p.cnp[p.loc[o]], 1); atomicMin(&p.ckey[p.loc[o]], res_depth_key(p, q)); }
    }
    sync();
    carry = 0;
    for (int base = 0; base < ncomp; base += GNT) {
        const int c = base + gtid;
        int tot;
        const int off = scan(c < ncomp ? p.cnp[c] : 0, tot);
        if (c < ncomp) p.cstart[c] = carry + off;
        carry += tot;
    }
    sync();
    for (int q = gtid; q < np; q += GNT) {
        const int o = res_owner(p, q, p.label);
        if (o < 0) continue;
        const int c = p.loc[o];
        p.cq[p.cstart[c] + atomicAdd(&p.cfill[c], 1)] = q;
    }
    sync();
    // a detached body's system: its own pairs (cfill of them, in cq) and the pairs of its partners' components;
    // cnp = the total, which decides the class
    for (int c = gtid; c < ncomp; c += GNT) {
        int tot = p.cnp[c], key = p.ckey[c];
        const int own = p.cown[c];
        if (own >= 0) {
            const int ps = p.cstart[c], no = p.cfill[c];
            for (int k = 0; k < no; ++k) {
                const int q = p.cq[ps + k];
                const int h = p.pairs[2 * q] == own ? p.pairs[2 * q + 1] : p.pairs[2 * q];
                const int cc = p.aux[h];
                if (cc < 0) continue;
                bool seen = false;
                for (int m = 0; m < k; ++m) {
                    const int q2 = p.cq[ps + m];
                    const int h2 = p.pairs[2 * q2] == own ? p.pairs[2 * q2 + 1] : p.pairs[2 * q2];
                    seen |= p.aux[h2] == cc;
                }
                if (!seen) { tot += p.cfill[cc]; key = min(key, p.ckey[cc]); }
            }
        }
        p.cnp[c] = tot;
        int cls = res_class(tot);
        if (cls == 5 && key < __float_as_int(RES_DEEP_RATIO))              // scheduling only: the long chains first, by depth
            cls = key < __float_as_int(RES_DEEP_RATIO / 64.f) ? 6 : key < __float_as_int(RES_DEEP_RATIO / 16.f) ? 7 : key < __float_as_int(RES_DEEP_RATIO / 4.f) ? 8 : 9;
        p.clist[(size_t)cls * p.cap + atomicAdd(&p.ctl[RES_CTL_CNT + cls], 1)] = c;
    }
    sync();
    if (gtid == 0) {
        p.ctl[0] = ncomp;
        p.mode[1] = (p.ctl[RES_CTL_CNT + 1] + p.ctl[RES_CTL_CNT + 2] + p.ctl[RES_CTL_CNT + 3] + p.ctl[RES_CTL_CNT + 4]) > 0 ? 1 : 0;
    }
}

// reciprocal square root to ~2 ulp: MUFU seed (22 bits) and one third-order correction (truncation 5/16 e^3 < 1e-19)
__device__ __forceinline__ double res_rsqrt(double a) {
    const double y = rsqrt_seed(a);
    const double e = fma(-a, y * y, 1.0);
    return fma(y, e * fma(0.375, e, 0.5), y);
}

// (1 - K(r; rc)) / r^3 with K the changeover weight of readings A-1..A-5 (rc2 = rc^2, inv = 1 / (0.9 rc)):
// 0 outside rc, 1/r^3 inside 0.1 rc; coincident bodies contribute 0 (X-5)
__device__ __forceinline__ double res_pair_u(double s2, double rc2, double inv) {
    if (!(s2 < rc2) || !(s2 > 0.0)) return 0.0;
    const double y = res_rsqrt(s2);
    const double q = fmin(fma(s2 * y, inv, -1.0 / 9.0), 1.0);          // (r - 0.1 rc) / (0.9 rc)
    const double K = q > 0.0 ? q * q * q * fma(q, fma(6.0, q, -15.0), 10.0) : 0.0;
    return (1.0 - K) * (y * y * y);
}

// the same without a branch (the small systems' kernel: one warp, straight-line code)
__device__ __forceinline__ double res_pair_u_nb(double s2, double rc2, double inv) {
    const bool in = (s2 < rc2) && (s2 > 0.0);
    const double y = res_rsqrt(in ? s2 : 1.0);
    const double q = fmin(fma(s2 * y, inv, -1.0 / 9.0), 1.0);
    const double K = q > 0.0 ? q * q * q * fma(q, fma(6.0, q, -15.0), 10.0) : 0.0;
    const double r = (1.0 - K) * (y * y * y);
    return in ? r : 0.0;
}

// ---- controller (uniform over the CTA: every thread takes the same decisions from the same block-wide numbers) ----
// Column k (n_k = 2 (k + 1) substeps) has the error estimate err_k = max |T_kk - T_k,k-1| / scale ~ H^(2k+1); the step
// that would make column k just converge is H_k = H fac_k, fac_k = 0.94 (0.65 tol / err_k)^(1/(2k+1)), and its work
// per unit step W_k = A_k / H_k with A_k = right-hand sides up to column k.  A step is accepted at the first column
// whose error is below tol; the next step aims at the column with the least work per unit step (one column down if
// W_k-1 < 0.9 W_k, one up if W_k < 0.9 W_k-1).  Columns up to target + 1 are tried, with the usual early exits when
// convergence cannot be expected; a rejected step is retried with H fac_k (at most 0.7 H).  40 rejections in a row
// are a failure: the component keeps its Kepler-drift result and is counted.
__device__ __forceinline__ float res_fac(double e, int k) {
    if (!(e > 0.0)) return 4.0f;
    const float r = 0.94f * exp2f(__log2f(0.65f / (float)fmin(e, 1e30)) / (float)(2 * k + 1));
    return fminf(fmaxf(r, 0.02f), 4.0f);
}
__device__ __forceinline__ double res_work(int k) { return (double)(k * k + 3 * k + 3); }   // 1 + sum_{j<=k} 2 (j + 1)
__device__ __forceinline__ bool res_hopeless(double e, int k, int ktarg) {
    if (k == ktarg - 1) { const double r = (double)((k + 2) * (k + 3)); return e > r * r; }     // (n_k+1 n_k+2 / n_0^2)^2
    if (k == ktarg) { const double r = (double)(k + 2); return e > r * r; }                     // (n_k+1 / n_0)^2
    return false;
}
struct ResCtl {
    double H;
    int ktarg, rejects;
    __device__ __forceinline__ void accepted(int acc, float facCur, float facPrev) {
        const double Wk = res_work(acc) / facCur, Wkm = acc >= 2 ? res_work(acc - 1) / facPrev : 1e300;
        int knew = acc;
        double hf = facCur;
        if (acc >= 2 && Wkm < 0.9 * Wk) { knew = acc - 1; hf = facPrev; }
        else if (acc < RES_KMAX - 1 && (acc < 2 || Wk < 0.9 * Wkm)) { knew = acc + 1; hf = facCur * (res_work(acc + 1) / res_work(acc)); }
        ktarg = max(2, min(knew, RES_KMAX - 1));
        H *= fmin(hf, 4.0);
        rejects = 0;
    }
    __device__ __forceinline__ bool rejected(int klast, float facLast) {    // true: give up
        H *= fminf(facLast, 0.7f);
        ktarg = max(2, min(ktarg, klast));
        return ++rejects > 40;
    }
};

// One CTA per component of class CLS, one thread per body (n <= np + 1 <= NT).  Shared memory, carved by the
// component's actual size: the pair region (87 B per pair), the body region (129 B per body: increments, y, f(y),
// inverse error scales, adjacency ranges) and - when it still fits - the extrapolation tableau (384 B per body),
// else global scratch.  Registers hold only the two running increments of the midpoint rule.  Only the warps that
// hold a body (nact = n rounded up to whole warps) run the Bulirsch-Stoer loop, synchronised by a named barrier of
// nact threads; the others wait at the block barrier that ends the component.
template <int NT, int CLS, int NCOL>
__global__ void __launch_bounds__(NT, 1) resolve_solve_kernel(ResParams p, int smemBytes) {
    extern __shared__ __align__(16) unsigned char res_dyn[];
    __shared__ double sRed[32];
    __shared__ int sScan[64];
    __shared__ int sBc[2];
    // SLICE (classes 1 and 2): the columns of a step stay in the shared memory of the CTAs that integrated them, and the
    // extrapolation tableau is SHARED OUT - CTA c runs it for the bodies [c S, (c + 1) S), S = n / NCOL, reading the
    // columns from the other CTAs' shared memory (distributed shared memory, ~0.1 us a load), and every CTA fetches the
    // row maxima of the error estimates and, after an accepted step, its bodies' increments from their owners.  Measured
    // on Jupiter's star at cfg3 (342 bodies, 92 attempted steps; per attempt, longest column 22 us): with the results in
    // global memory and the whole tableau in every CTA the exchange cost 5 + 14 us per attempt (profiles/r2d_resolve.md).
    // The slice's tableau is in shared memory when there is room (always, up to 512 bodies), else in global scratch.
    constexpr bool SLICE = NCOL > 1;
    __shared__ double sRedK[SLICE ? 4 : 1][RES_KMAX];                      // the slice warps' error maxima of every tableau row
    __shared__ double sErr[RES_KMAX];                                      // this CTA's slice: error maximum of every row
    __shared__ int sStop;                                                  // the cluster-barrier phase after which the warps without a body leave
    constexpr unsigned full = 0xffffffffu;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid < 64) sScan[tid] = 0;
    bool firstTicket = true;
    // NCOL > 1: the NCOL CTAs of a thread-block cluster work on the same component, CTA `col` integrating column `col` of
    // every Bulirsch-Stoer step (the columns - 2, 4, .., 16 substeps from the same state - are independent integrations:
    // side by side a step costs its longest column instead of their sum); components dealt to the clusters round-robin
    const int col = NCOL > 1 ? (int)(blockIdx.x % NCOL) : 0;
    const int cl = blockIdx.x / NCOL, ncl = gridDim.x / NCOL;
    int round = 0;

    for (;;) {
    __syncthreads();                                                       // the previous component is finished with shared memory
    if (SLICE && tid == 0) sStop = 0x7fffffff;
    int ticket;
    if (NCOL > 1) ticket = cl + (round++) * ncl;
    else if (firstTicket) { ticket = blockIdx.x; firstTicket = false; }    // the first gridDim.x components need no counter
    else {
        if (tid == 0) sBc[0] = gridDim.x + atomicAdd(&p.ctl[RES_CTL_TKT + CLS], 1);
        __syncthreads();
        ticket = sBc[0];
    }
    if (ticket >= p.ctl[RES_CTL_CNT + CLS]) break;
    const int comp = p.clist[(size_t)CLS * p.cap + ticket];
    const int np = p.cnp[comp];
    const int npad = SLICE ? (np + 32) & ~31 : (np + 31) & ~31;             // (SLICE: at least as many slots as bodies - sF doubles as the column result)
    double* const sF = reinterpret_cast<double*>(res_dyn);                  // [3][npad] pair terms
    double* const sDy = sF + 3 * npad;                                      // [3][npad] y_j - y_i of the state the BS step starts from
    double* const sRc2 = sDy + 3 * npad;                                    // [npad] max(rcrit_i, rcrit_j)^2
    double* const sInv = sRc2 + npad;                                       // [npad] 1 / (0.9 rc)
    double* const sGi = sInv + npad;                                        // [npad] gm of the first member
    double* const sGj = sGi + npad;                                         // [npad] gm of the second member
    unsigned short* const sPi = reinterpret_cast<unsigned short*>(sGj + npad);   // [npad] local members of each pair
    unsigned short* const sPj = sPi + npad;
    unsigned short* const sAdj = sPj + npad;                                // [npad] pairs of each body as second member, list order
    double* const sGs = reinterpret_cast<double*>(sAdj + npad);             // [3][npad / 32] a hub's terms summed over whole groups of 32 pairs
    const int pairBytes = (86 * npad + 24 * (npad >> 5) + 15) & ~15;
    int* const tQ = reinterpret_cast<int*>(sF);                             // setup only, on the 48 npad bytes of sF and sDy:
    int* const tQs = tQ + npad;                                             // 4 npad ints + the body list (npad + 32 ints) [+ 4 npad ints]
    int* const tBi = tQs + npad;
    int* const tBj = tBi + npad;
    int* const tBody = tBj + npad;

    // ---- the component's pairs in list order (the label kernel grouped them in arrival order: rank sort) ----
    const int own = p.cown[comp];                                          // a detached body's system (see res_owner), else -1
    {
        const int ps = p.cstart[comp], nown = p.cfill[comp];
        for (int k = tid; k < nown; k += NT) tQ[k] = p.cq[ps + k];
        __syncthreads();
        if (own >= 0 && tid == 0) {                                        // + the pairs of its partners' components, each once
            int cnt = nown;
            for (int k = 0; k < nown; ++k) {
                const int q = tQ[k];
                const int cc = p.aux[p.pairs[2 * q] == own ? p.pairs[2 * q + 1] : p.pairs[2 * q]];
                if (cc < 0) continue;
                bool seen = false;
                for (int m = 0; m < k; ++m) { const int q2 = tQ[m]; seen |= p.aux[p.pairs[2 * q2] == own ? p.pairs[2 * q2 + 1] : p.pairs[2 * q2]] == cc; }
                if (!seen) for (int m = 0; m < p.cfill[cc]; ++m) tQ[cnt++] = p.cq[p.cstart[cc] + m];
            }
        }
        __syncthreads();
#pragma unroll 1
        for (int k = tid; k < np; k += NT) {
            const int mine = tQ[k];
            int r = 0;
#pragma unroll 4
            for (int m = 0; m < np; ++m) r += (tQ[m] < mine) ? 1 : 0;
            tQs[r] = mine;
        }
        __syncthreads();
    }
    // ---- its bodies, numbered by first appearance in the list (deterministic) ----
    // no shared body -> index table: a detached body's partners are in other systems too, and the CTAs of a cluster set
    // the same component up side by side
    const bool search = own >= 0 || NCOL > 1;
    int* const tFirst = tBody + npad + 32;                                  // search only: 2 npad + 2 npad more ints
    int* const tId = tFirst + 2 * npad;
#pragma unroll 1
    for (int k = tid; k < np; k += NT) {
        const int q = tQs[k], bi = p.pairs[2 * q], bj = p.pairs[2 * q + 1];
        tBi[k] = bi; tBj[k] = bj;
        if (!search) { p.loc[bi] = 0x7fffffff; p.loc[bj] = 0x7fffffff; }
    }
    __syncthreads();
    int n = 0;
    if (!search) {
        // a component's bodies are in no other component: the global body -> index table is theirs alone
#pragma unroll 1
        for (int k = tid; k < np; k += NT) { atomicMin(&p.loc[tBi[k]], 2 * k); atomicMin(&p.loc[tBj[k]], 2 * k + 1); }
        __syncthreads();
#pragma unroll 1
        for (int base = 0; base < np; base += NT) {
            const int k = base + tid;
            int fi = 0, fj = 0;
            if (k < np) { fi = (p.loc[tBi[k]] == 2 * k) ? 1 : 0; fj = (p.loc[tBj[k]] == 2 * k + 1) ? 1 : 0; }
            int tot;
            const int off = res_scan(fi + fj, sScan, tot);
            if (fi) tBody[n + off] = tBi[k];
            if (fj) tBody[n + off + fi] = tBj[k];
            n += tot;
        }
    } else {
        // a detached body's massive partners are also in the systems of their other test particles (and perhaps in a
        // component): no shared table - first appearances by search in the system's own (short) list
#pragma unroll 1
        for (int pos = tid; pos < 2 * np; pos += NT) {
            const int b = (pos & 1) ? tBj[pos >> 1] : tBi[pos >> 1];
            int f = pos;
            for (int m = pos - 1; m >= 0; --m) if (((m & 1) ? tBj[m >> 1] : tBi[m >> 1]) == b) f = m;
            tFirst[pos] = f;
        }
        __syncthreads();
#pragma unroll 1
        for (int base = 0; base < 2 * np; base += NT) {
            const int pos = base + tid;
            const int isf = (pos < 2 * np && tFirst[pos] == pos) ? 1 : 0;
            int tot;
            const int off = res_scan(isf, sScan, tot);
            if (isf) { tId[pos] = n + off; tBody[n + off] = (pos & 1) ? tBj[pos >> 1] : tBi[pos >> 1]; }
            n += tot;
        }
    }
    __syncthreads();
    const int nbp = (n + 31) & ~31;
    double* const sP = reinterpret_cast<double*>(res_dyn + pairBytes);      // [3][nbp] increments z - y of the current right-hand side (y for f(y))
    double* const sY = sP + 3 * nbp;                                        // [6][nbp] state at the start of the BS step
    double* const sF0 = sY + 6 * nbp;                                       // [3][nbp] acceleration there
    double* const sIS = sF0 + 3 * nbp;                                      // [2][nbp] 1 / |x|, 1 / |v| there (error scales)
    int* const sILo = reinterpret_cast<int*>(sIS + 2 * nbp);                // [nbp] pairs of a body as first member: [iLo, iHi)
    int* const sIHi = sILo + nbp;
    int* const sD2 = sIHi + nbp;                                            // [nbp] number of pairs as second member
    int* const sJLo = sD2 + nbp;                                            // [nbp] their first slot in sAdj
    unsigned char* const sHv = reinterpret_cast<unsigned char*>(sJLo + nbp);   // [nbp] 1: a hub (more than RES_HEAVY pairs)
    const int bodyBytes = 129 * nbp + 15 & ~15;
    const bool live = tid < n;
    const int me = live ? tBody[tid] : 0;
    if (live) { if (!search) p.loc[me] = tid; sILo[tid] = 0; sIHi[tid] = 0; sD2[tid] = 0; }
    __syncthreads();
#pragma unroll 1
    for (int k = tid; k < np; k += NT) {
        const int bi = tBi[k], bj = tBj[k];
        const int li = !search ? p.loc[bi] : tId[tFirst[2 * k]], lj = !search ? p.loc[bj] : tId[tFirst[2 * k + 1]];
        sPi[k] = (unsigned short)li; sPj[k] = (unsigned short)lj;
        sGi[k] = p.gm[bi]; sGj[k] = p.gm[bj];
        const double rc = fmax(p.rcrit[bi], p.rcrit[bj]);
        sRc2[k] = rc * rc; sInv[k] = rc > 0.0 ? 1.0 / (0.9 * rc) : 0.0;
        if (k == 0 || tBi[k - 1] != bi) sILo[li] = k;                       // the list is sorted by (i, j): one run per first member
        if (k == np - 1 || tBi[k + 1] != bi) sIHi[li] = k + 1;
        atomicAdd(&sD2[lj], 1);
    }
    __syncthreads();
    {
        int tot;
        const int off = res_scan(live ? sD2[tid] : 0, sScan, tot);
        if (live) sJLo[tid] = off;
    }
    __syncthreads();
#pragma unroll 1
    for (int k = tid; k < np; k += NT) {
        const int lj = sPj[k];
        int r = 0;
        if (sD2[lj] > 1) for (int m = 0; m < k; ++m) r += (sPj[m] == lj) ? 1 : 0;
        sAdj[sJLo[lj] + r] = (unsigned short)k;
    }
    const int iLo = live ? sILo[tid] : 0, iHi = live ? sIHi[tid] : 0, jLo = live ? sJLo[tid] : 0, d2 = live ? sD2[tid] : 0;
    const bool heavy = d2 + iHi - iLo > RES_HEAVY;
    if (tid < nbp) {
        sHv[tid] = heavy ? 1 : 0;
#pragma unroll
        for (int c = 0; c < 3; ++c) {                                      // pad rows: a harmless body at (1, 0, 0)
            sY[c * nbp + tid] = live ? p.x0[(size_t)c * p.ld + me] : (c == 0 ? 1.0 : 0.0);
            sY[(3 + c) * nbp + tid] = live ? p.v0[(size_t)c * p.ld + me] : 0.0;
        }
    }
    for (int k = np + tid; k < npad; k += NT) sPi[k] = 0xffff;              // pad pairs: no group of theirs is a whole run of a hub
    __syncthreads();                                                       // the temporaries (on sF, sDy) are consumed; sAdj is complete
    const int S = nbp / (NCOL > 1 ? NCOL : 1);                              // SLICE: bodies of the tableau slice of a CTA (nbp is a multiple of 32)
    const int SLW = (S + 31) & ~31;                                         // ... and the threads (whole warps) that work on it
    // SLICE: [6 KMAX][S] tableau of this CTA's slice - in shared memory when there is room (always, up to 512 bodies), else in
    // this CTA's part of the global scratch (the cluster's barrier orders its writes before the other CTAs' ld.cg reads)
    // (known at compile time for the classes up to 512 threads: plain shared-memory addressing there)
    const bool sliceShared = NT <= 512 || pairBytes + bodyBytes + 6 * RES_KMAX * 8 * S <= smemBytes;
    double* const sT = reinterpret_cast<double*>(res_dyn + pairBytes + bodyBytes);
    double* const gT = p.tab + (size_t)blockIdx.x * 6 * RES_KMAX * NT;
    const bool tabShared = pairBytes + bodyBytes + 6 * RES_KMAX * 8 * nbp <= smemBytes;
    const int TS = tabShared ? nbp : NT;                                    // tableau stride
    double* const Tb = (tabShared ? reinterpret_cast<double*>(res_dyn + pairBytes + bodyBytes)
                                  : p.tab + (size_t)blockIdx.x * 6 * RES_KMAX * NT) + tid;   // T_{row, j}, component c of this body at Tb[(j * 6 + c) * TS]

    // ---- the Bulirsch-Stoer loop ----
    // Right-hand side at the positions y + dl (ONE inlined copy: f(y) itself is the iteration m = 0 of the first column
    // after an accepted step).  The separations of the listed pairs are formed as (y_j - y_i) + (dl_j - dl_i) with the
    // first bracket taken once per BS step (m = 0: dl = 0, the bracket is stored): the stages of a step then differ by
    // exactly rounded small numbers instead of by the rounding of AU-sized sums, whose noise (eps |x| / r relative,
    // amplified by the extrapolation) would otherwise sit above a tolerance of 1e-12 during a close passage.
    const int nact = nbp;                                                  // threads of the warps that hold a body
    if (tid < nact) {
    const double mu = p.mu, hh = p.h, tol = p.tol;
    double t = 0.0;
    ResCtl ctl{hh, 5, 0};
    int fail = 0, nacc = 0, nrhs = 0;
    int nphase = 0;                                                        // SLICE: phases of the cluster barrier passed in this component
    bool havef0 = false;
    while (!fail) {
        const double rem = hh - t;
        if (fabs(rem) <= 4.0 * 2.220446049250313e-16 * fabs(hh)) break;
        bool last = false;
        if (fabs(ctl.H) >= fabs(rem)) { ctl.H = rem; last = true; }
        const double H = ctl.H;
        const int kcols = min(ctl.ktarg + 1, RES_KMAX - 1);
        int acc = -1, klast = 0;
        float facCur = 1.0f, facPrev = 1.0f;
        // column kk: the modified midpoint rule with 2 (kk + 1) substeps over H -> cur (its increment); with run = false only
        // f(y) and the error scales (m = 0), when they are still missing
        auto column = [&](const int kk, const bool run, double (&cur)[6]) {
            const int nsub = 2 * (kk + 1);
            const double hs = H / (double)nsub;
            double d0[6], d1[6];
#pragma unroll
            for (int c = 0; c < 6; ++c) { d0[c] = 0.0; d1[c] = 0.0; cur[c] = 0.0; }
            if (havef0 && live) {
#pragma unroll
                for (int c = 0; c < 3; ++c) { d1[c] = hs * sY[(3 + c) * nbp + tid]; d1[3 + c] = hs * sF0[c * nbp + tid]; }
            }
            const int mlast = run ? nsub : 0;
#pragma unroll 1
            for (int m = havef0 ? 1 : 0; m <= mlast; ++m) {
                const bool base = m == 0;
                // own position: the increment goes to shared memory (y itself for f(y))
                const double y0 = sY[tid], y1 = sY[nbp + tid], y2 = sY[2 * nbp + tid];
                const double v0 = sY[3 * nbp + tid] + d1[3], v1 = sY[4 * nbp + tid] + d1[4], v2 = sY[5 * nbp + tid] + d1[5];
                sP[tid] = base ? y0 : d1[0]; sP[nbp + tid] = base ? y1 : d1[1]; sP[2 * nbp + tid] = base ? y2 : d1[2];
                res_bar(nact);
                // star's Kepler term and the first pair of this thread in one straight line (two independent chains)
                const double z0 = y0 + d1[0], z1 = y1 + d1[1], z2 = y2 + d1[2];            // d1 = 0 when base
                const double yk = res_rsqrt(fma(z2, z2, fma(z1, z1, z0 * z0)));
                const double wk = -mu * (yk * yk * yk);
                double a0 = wk * z0, a1 = wk * z1, a2 = wk * z2;
#pragma unroll 1
                for (int q = tid; q < np; q += nact) {
                    const int i = sPi[q], j = sPj[q];
                    double dx = sP[j] - sP[i], dy = sP[nbp + j] - sP[nbp + i], dz = sP[2 * nbp + j] - sP[2 * nbp + i];
                    if (base) { sDy[q] = dx; sDy[npad + q] = dy; sDy[2 * npad + q] = dz; }
                    else { dx += sDy[q]; dy += sDy[npad + q]; dz += sDy[2 * npad + q]; }
                    const double u = res_pair_u(fma(dz, dz, fma(dy, dy, dx * dx)), sRc2[q], sInv[q]);
                    const double f0 = u * dx, f1 = u * dy, f2 = u * dz;
                    sF[q] = f0; sF[npad + q] = f1; sF[2 * npad + q] = f2;
                    // a whole group of 32 pairs with the same hub as first member: its sum by a shuffle tree now, in
                    // every warp at once, instead of term by term in the hub's warp afterwards
                    const int ia = sPi[q & ~31];
                    if (ia == sPi[q | 31] && sHv[ia]) {                     // warp-uniform
                        const double g = sGj[q];
                        double h0 = g * f0, h1 = g * f1, h2 = g * f2;
#pragma unroll
                        for (int o = 16; o > 0; o >>= 1) {
                            h0 += __shfl_xor_sync(full, h0, o); h1 += __shfl_xor_sync(full, h1, o); h2 += __shfl_xor_sync(full, h2, o);
                        }
                        if (lane == 0) { const int g5 = q >> 5, ng = npad >> 5; sGs[g5] = h0; sGs[ng + g5] = h1; sGs[2 * ng + g5] = h2; }
                    }
                }
                res_bar(nact);
                unsigned hm = __ballot_sync(full, heavy);
                while (hm) {                                               // a hub: its warp sums together
                    const int l = __ffs(hm) - 1;
                    hm &= hm - 1;
                    const int j0 = __shfl_sync(full, jLo, l), dj = __shfl_sync(full, d2, l);
                    const int i0 = __shfl_sync(full, iLo, l), i1 = __shfl_sync(full, iHi, l);
                    double h0 = 0.0, h1 = 0.0, h2 = 0.0;
#pragma unroll 1
                    for (int e = lane; e < dj; e += 32) {                  // the hub as second member: -gm_i u d
                        const int q = sAdj[j0 + e];
                        const double g = sGi[q];
                        h0 = fma(-g, sF[q], h0); h1 = fma(-g, sF[npad + q], h1); h2 = fma(-g, sF[2 * npad + q], h2);
                    }
                    // as first member: +gm_j u d - whole groups from their sums, the ragged ends term by term
                    const int gA = (i0 + 31) >> 5, gB = i1 >> 5, ng = npad >> 5;
                    const int qa = gA < gB ? gA << 5 : i1, qb = gA < gB ? gB << 5 : i1;    // [i0, qa) and [qb, i1) term by term
#pragma unroll 1
                    for (int g5 = gA + lane; g5 < gB; g5 += 32) { h0 += sGs[g5]; h1 += sGs[ng + g5]; h2 += sGs[2 * ng + g5]; }
#pragma unroll 1
                    for (int q = i0 + lane; q < qa; q += 32) {
                        const double g = sGj[q];
                        h0 = fma(g, sF[q], h0); h1 = fma(g, sF[npad + q], h1); h2 = fma(g, sF[2 * npad + q], h2);
                    }
#pragma unroll 1
                    for (int q = qb + lane; q < i1; q += 32) {
                        const double g = sGj[q];
                        h0 = fma(g, sF[q], h0); h1 = fma(g, sF[npad + q], h1); h2 = fma(g, sF[2 * npad + q], h2);
                    }
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) {
                        h0 += __shfl_xor_sync(full, h0, o); h1 += __shfl_xor_sync(full, h1, o); h2 += __shfl_xor_sync(full, h2, o);
                    }
                    if (lane == l) { a0 += h0; a1 += h1; a2 += h2; }
                }
                if (live && !heavy) {
#pragma unroll 1
                    for (int e = jLo; e < jLo + d2; ++e) {
                        const int q = sAdj[e];
                        const double g = sGi[q];
                        a0 = fma(-g, sF[q], a0); a1 = fma(-g, sF[npad + q], a1); a2 = fma(-g, sF[2 * npad + q], a2);
                    }
#pragma unroll 1
                    for (int q = iLo; q < iHi; ++q) {
                        const double g = sGj[q];
                        a0 = fma(g, sF[q], a0); a1 = fma(g, sF[npad + q], a1); a2 = fma(g, sF[2 * npad + q], a2);
                    }
                }
                ++nrhs;
                if (base) {                                                // f(y) and the error scales of this BS step
                    if (live) {
                        sF0[tid] = a0; sF0[nbp + tid] = a1; sF0[2 * nbp + tid] = a2;
                        const double sx2 = fma(y2, y2, fma(y1, y1, y0 * y0)), sv2 = fma(v2, v2, fma(v1, v1, v0 * v0));
                        sIS[tid] = sx2 > 0.0 ? 1.0 / sqrt(sx2) : 1e300; sIS[nbp + tid] = sv2 > 0.0 ? 1.0 / sqrt(sv2) : 1e300;
                        d1[0] = hs * v0; d1[1] = hs * v1; d1[2] = hs * v2; d1[3] = hs * a0; d1[4] = hs * a1; d1[5] = hs * a2;
                    }
                    havef0 = true;
                } else if (m < nsub) {
                    const double h2s = 2.0 * hs;
                    double tt;
                    tt = fma(h2s, v0, d0[0]); d0[0] = d1[0]; d1[0] = tt;
                    tt = fma(h2s, v1, d0[1]); d0[1] = d1[1]; d1[1] = tt;
                    tt = fma(h2s, v2, d0[2]); d0[2] = d1[2]; d1[2] = tt;
                    tt = fma(h2s, a0, d0[3]); d0[3] = d1[3]; d1[3] = tt;
                    tt = fma(h2s, a1, d0[4]); d0[4] = d1[4]; d1[4] = tt;
                    tt = fma(h2s, a2, d0[5]); d0[5] = d1[5]; d1[5] = tt;
                } else {
                    cur[0] = 0.5 * (d0[0] + fma(hs, v0, d1[0])); cur[1] = 0.5 * (d0[1] + fma(hs, v1, d1[1])); cur[2] = 0.5 * (d0[2] + fma(hs, v2, d1[2]));
                    cur[3] = 0.5 * (d0[3] + fma(hs, a0, d1[3])); cur[4] = 0.5 * (d0[4] + fma(hs, a1, d1[4])); cur[5] = 0.5 * (d0[5] + fma(hs, a2, d1[5]));
                }
            }
        };
        if constexpr (SLICE) {
            // Every CTA its own column (the CTAs beyond the columns this step tries: f(y) only).  The result goes where the
            // right-hand side's scratch was - rows 0..2 on sP, rows 3..5 on sF (npad >= nbp) - for the other CTAs to read.
            // Two phases of the cluster's hardware barrier per step: A - the columns are there; B - the slices' tableaux
            // and error maxima are there, and nobody reads a column any more.  Whoever writes the next column, tableau
            // or maxima has passed the barrier all their readers arrive at only after reading.
            double mine[6];
            column(col, col <= kcols, mine);
            res_bar(nact);                                                 // the last right-hand side's sums have read sF
            if (live && col <= kcols) {
#pragma unroll
                for (int c = 0; c < 3; ++c) { sP[c * nbp + tid] = mine[c]; sF[c * npad + tid] = mine[3 + c]; }
            }
            res_cl_sync(); ++nphase;                                       // A
            if (col == 0) nrhs += (kcols + 1) * (kcols + 2) - 2;            // the other columns' right-hand sides: sum of 2 (k + 1)
            if (tid < SLW) {
                // this CTA's slice of the tableau: body b, rows 0..kcols in place (entry j * 6 + c at sT[(j * 6 + c) S + tid];
                // row k's column comes from CTA k, the next row's is on its way while this row is extrapolated)
                const int b = col * S + tid;
                const bool liveS = tid < S && b < n;
                const int bb = liveS ? b : 0;
                double nxt[6];
#pragma unroll
                for (int c = 0; c < 3; ++c) { nxt[c] = res_ld_remote(&sP[c * nbp + bb], 0); nxt[3 + c] = res_ld_remote(&sF[c * npad + bb], 0); }
                const double isx = sIS[bb], isv = sIS[nbp + bb];
                double* const T = (sliceShared ? sT : gT) + tid;
#pragma unroll 1
                for (int k = 0; k <= kcols; ++k) {
                    double cur[6], prev[6];
#pragma unroll
                    for (int c = 0; c < 6; ++c) { cur[c] = nxt[c]; prev[c] = cur[c]; }
                    if (k < kcols) {
#pragma unroll
                        for (int c = 0; c < 3; ++c) { nxt[c] = res_ld_remote(&sP[c * nbp + bb], k + 1); nxt[3 + c] = res_ld_remote(&sF[c * npad + bb], k + 1); }
                    }
                    double err = 0.0;
                    if (liveS) {
#pragma unroll 1
                        for (int j = 1; j <= k; ++j) {
                            const double cf = RES_COEF[k * RES_KMAX + j];
#pragma unroll
                            for (int c = 0; c < 6; ++c) {
                                double* tp = T + ((j - 1) * 6 + c) * S;
                                const double oldv = *tp;
                                *tp = cur[c];
                                prev[c] = cur[c];
                                cur[c] = fma(cur[c] - oldv, cf, cur[c]);
                            }
                        }
#pragma unroll
                        for (int c = 0; c < 6; ++c) {
                            T[(k * 6 + c) * S] = cur[c];
                            double e = fabs(cur[c] - prev[c]) * (c < 3 ? isx : isv);
                            if (!(e <= 1e300)) e = 1e300;                   // NaN / inf: never accepted
                            err = fmax(err, e);
                        }
                    }
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) err = fmax(err, __shfl_xor_sync(full, err, o));
                    if (lane == 0) sRedK[warp][k] = err;
                }
                asm volatile("bar.sync 2, %0;" ::"r"(SLW) : "memory");      // the slice's warps
                if (tid < RES_KMAX) {
                    double v = 0.0;
                    for (int w2 = 0; w2 < SLW / 32; ++w2) v = fmax(v, sRedK[w2][tid]);
                    sErr[tid] = tid <= kcols ? v : 0.0;
                }
            }
            res_cl_sync(); ++nphase;                                       // B
            // the rows' error maxima over all the slices: lane l reads rows (l >> 3) + 1 and (l >> 3) + 5 of CTA l & 7
            {
                const int r0 = (lane >> 3) + 1, r1 = (lane >> 3) + 5;
                double v0 = res_ld_remote(&sErr[r0], lane & (NCOL - 1));
                double v1 = r1 < RES_KMAX ? res_ld_remote(&sErr[r1], lane & (NCOL - 1)) : 0.0;
#pragma unroll
                for (int o = 4; o > 0; o >>= 1) { v0 = fmax(v0, __shfl_xor_sync(full, v0, o)); v1 = fmax(v1, __shfl_xor_sync(full, v1, o)); }
                bool done = false;
                double eL = 0.0, eP = 0.0;                                  // the error of the last row looked at, and of the one before
#pragma unroll
                for (int k = 1; k < RES_KMAX; ++k) {
                    const double e = (k <= 4 ? __shfl_sync(full, v0, (k - 1) * 8) : __shfl_sync(full, v1, (k - 5) * 8)) / tol;
                    if (k <= kcols && !done) {
                        eP = eL; eL = e; klast = k;
                        if (e <= 1.0) { acc = k; done = true; }
                        else if (k < kcols && res_hopeless(e, k, ctl.ktarg)) done = true;
                    }
                }
                facCur = res_fac(eL, klast);
                facPrev = klast >= 2 ? res_fac(eP, klast - 1) : 1.0f;
            }
            if (acc >= 0 && live) {                                        // this body's increment from the CTA that ran its tableau
                const int o = tid / S, i = tid - o * S;
#pragma unroll
                for (int c = 0; c < 6; ++c)
                    sY[c * nbp + tid] += sliceShared ? res_ld_remote(&sT[(acc * 6 + c) * S + i], o)
                                                     : __ldcg(&p.tab[((size_t)blockIdx.x - col + o) * 6 * RES_KMAX * NT + (size_t)(acc * 6 + c) * S + i]);
            }
        }
#pragma unroll 1
        for (int k = 0; !SLICE && k <= kcols; ++k) {
            double cur[6];
            column(k, true, cur);
            // row k of the tableau from row k-1 (in T), overwriting it column by column
            double err = 0.0;
            if (live) {
                double prev[6];
#pragma unroll
                for (int c = 0; c < 6; ++c) prev[c] = cur[c];
#pragma unroll 1
                for (int j = 1; j <= k; ++j) {
                    const double cf = RES_COEF[k * RES_KMAX + j];
#pragma unroll
                    for (int c = 0; c < 6; ++c) {
                        double* tp = Tb + (size_t)((j - 1) * 6 + c) * TS;
                        const double oldv = *tp;
                        *tp = cur[c];
                        prev[c] = cur[c];
                        cur[c] = fma(cur[c] - oldv, cf, cur[c]);
                    }
                }
                const double isx = sIS[tid], isv = sIS[nbp + tid];
#pragma unroll
                for (int c = 0; c < 6; ++c) {
                    Tb[(size_t)(k * 6 + c) * TS] = cur[c];
                    double e = fabs(cur[c] - prev[c]) * (c < 3 ? isx : isv);
                    if (!(e <= 1e300)) e = 1e300;                           // NaN / inf: never accepted
                    err = fmax(err, e);
                }
            }
            if (k >= 1) {
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) err = fmax(err, __shfl_xor_sync(full, err, o));
                if (lane == 0) sRed[warp] = err;
                res_bar(nact);
                double e = sRed[0];
#pragma unroll 1
                for (int w = 1; w < nact / 32; ++w) e = fmax(e, sRed[w]);
                e /= tol;
                facPrev = facCur; facCur = res_fac(e, k);
                klast = k;
                if (e <= 1.0) { acc = k; break; }
                if (k < kcols && res_hopeless(e, k, ctl.ktarg)) break;
            }
        }
        if (acc < 0) {
            if (ctl.rejected(klast, facCur)) fail = 1;
            continue;
        }
        if (!SLICE && live) {
#pragma unroll
            for (int c = 0; c < 6; ++c) sY[c * nbp + tid] += Tb[(size_t)(acc * 6 + c) * TS];
        }
        t = last ? hh : t + H;
        ++nacc;
        havef0 = false;
        ctl.accepted(acc, facCur, facPrev);
    }
    if constexpr (SLICE) {                                                 // one more phase, after which the warps without a body leave too
        if (tid == 0) sStop = nphase + 1;
        res_cl_sync();
    }
    if (!fail && live && col == 0 && (own < 0 || own == me)) {             // a detached body's system writes only that body
#pragma unroll
        for (int c = 0; c < 3; ++c) { p.x[(size_t)c * p.ld + me] = sY[c * nbp + tid]; p.v[(size_t)c * p.ld + me] = sY[(3 + c) * nbp + tid]; }
    }
    if (tid == 0 && col == 0) {
        atomicAdd(&p.out->bodies, own < 0 ? n : 1); atomicAdd(&p.out->steps, nacc); atomicAdd(&p.out->rhs, nrhs);
        if (fail) { atomicAdd(&p.out->fail, 1); atomicAdd(&p.st->resolve_fail, 1); }
    }
    }   // active warps
    else if constexpr (SLICE) {
        // the cluster's barrier counts every thread of its CTAs: the warps without a body go through its phases too
        for (int ph = 1;; ++ph) {
            res_cl_sync();
            if (ph == *reinterpret_cast<volatile int*>(&sStop)) break;
        }
    }
    }   // components
}

// ---- class S: the small systems (at most RES_PHI_S pairs, hence at most 32 bodies: a planetesimal pair, a test particle
// with its one or two big partners - almost every system of a list).  One CTA of RES_KMAX warps per system at a time, and
// the columns of a Bulirsch-Stoer step SIDE BY SIDE inside it: warp w integrates column w (2 (w + 1) substeps), lane =
// body for the state, lane = pair for the pair terms, everything in shared memory and registers, warp barriers only
// inside a right-hand side.  A step then costs its longest column (at most 17 right-hand sides) instead of the sum of
// its columns (42-72), and two block barriers: columns -> shared memory | warp 0 runs the extrapolation tableau and the
// error test, moves the state on acceptance and publishes the outcome | every warp updates the same controller from it.
// The deepest passage of a list - a test particle grazing an embryo: ~100 steps - is the length of the whole solve
// when the systems are many and small (N = 1e6, nbig = 100), which is why it is cut here and not the throughput.
// Same arithmetic and the same summation order per body (pairs as second member first, list order) as
// resolve_solve_kernel; the controller is the same code on the same numbers.
#ifndef RES_S_MINB
#define RES_S_MINB 2
#endif
__global__ void __launch_bounds__(RES_S_THREADS, RES_S_MINB) resolve_small_kernel(ResParams p) {
    constexpr int W = RES_KMAX;
    __shared__ double sY[6][32];                 // state at the start of the Bulirsch-Stoer step
    __shared__ double sP[W][3][32];              // per column: position increments of the current right-hand side (y for f(y))
    __shared__ double sFt[W][3][32];             // per column: pair terms
    __shared__ double sDy[W][3][32];             // per column (identical copies): y_j - y_i at the start of the step
    __shared__ double sCol[W][6][32];            // column results; warp 0 turns them into the extrapolation tableau in place
    __shared__ double sC[32][32];                // [pair][body]: +gm_j if the body is the pair's first member, -gm_i if its second, else 0
    __shared__ double sRc2[32], sInv[32], sGi[32], sGj[32];
    __shared__ int sPi[32], sPj[32], sQ[32], sQs[32], sBi[32], sBj[32], sBody[32], sFirst[64], sId[64];
    __shared__ float sFac[2];
    __shared__ int sCtl[4];                      // ticket | accepted column (-1: none) | last column tested | bodies
    constexpr unsigned full = 0xffffffffu;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const unsigned lt = (1u << lane) - 1u;
    bool firstTicket = true;

    for (;;) {
    __syncthreads();                                                       // the previous system is finished with shared memory
    int ticket;
    if (firstTicket) { ticket = blockIdx.x; firstTicket = false; }
    else {
        if (tid == 0) sCtl[0] = gridDim.x + atomicAdd(&p.ctl[RES_CTL_TKT + 5], 1);
        __syncthreads();
        ticket = sCtl[0];
    }
    int cls = 6, tk = ticket;                                              // the systems that look deep first, deepest first
    while (cls <= 9 && tk >= p.ctl[RES_CTL_CNT + cls]) { tk -= p.ctl[RES_CTL_CNT + cls]; ++cls; }
    if (cls > 9) { cls = 5; if (tk >= p.ctl[RES_CTL_CNT + 5]) break; }
    const int comp = p.clist[(size_t)cls * p.cap + tk];
    const int np = p.cnp[comp];
    const int own = p.cown[comp];                                          // a detached body's system (see res_owner), else -1

    // ---- set-up by warp 0: pairs in list order, bodies numbered by first appearance (as in resolve_solve_kernel) ----
    if (w == 0) {
        const int ps = p.cstart[comp], nown = p.cfill[comp];
        if (lane < nown) sQ[lane] = p.cq[ps + lane];
        __syncwarp();
        if (own >= 0 && lane == 0) {                                       // + the pairs of its partners' components, each once
            int cnt = nown;
            for (int k = 0; k < nown; ++k) {
                const int q = sQ[k];
                const int cc = p.aux[p.pairs[2 * q] == own ? p.pairs[2 * q + 1] : p.pairs[2 * q]];
                if (cc < 0) continue;
                bool seen = false;
                for (int m = 0; m < k; ++m) { const int q2 = sQ[m]; seen |= p.aux[p.pairs[2 * q2] == own ? p.pairs[2 * q2 + 1] : p.pairs[2 * q2]] == cc; }
                if (!seen) for (int m = 0; m < p.cfill[cc]; ++m) sQ[cnt++] = p.cq[p.cstart[cc] + m];
            }
        }
        __syncwarp();
        if (lane < np) {
            const int mine = sQ[lane];
            int r = 0;
            for (int m = 0; m < np; ++m) r += (sQ[m] < mine) ? 1 : 0;
            sQs[r] = mine;
        }
        __syncwarp();
        int bi = 0, bj = 0;
        if (lane < np) { const int q = sQs[lane]; bi = p.pairs[2 * q]; bj = p.pairs[2 * q + 1]; sBi[lane] = bi; sBj[lane] = bj; }
        __syncwarp();
        int isf0 = 0, isf1 = 0;
        if (lane < np) {
            int f0 = 2 * lane, f1 = 2 * lane + 1;
            for (int m = 2 * lane - 1; m >= 0; --m) if (((m & 1) ? sBj[m >> 1] : sBi[m >> 1]) == bi) f0 = m;
            for (int m = 2 * lane; m >= 0; --m) if (((m & 1) ? sBj[m >> 1] : sBi[m >> 1]) == bj) f1 = m;
            sFirst[2 * lane] = f0; sFirst[2 * lane + 1] = f1;
            isf0 = f0 == 2 * lane; isf1 = f1 == 2 * lane + 1;
        }
        const unsigned b0 = __ballot_sync(full, isf0), b1 = __ballot_sync(full, isf1);
        const int id0 = __popc(b0 & lt) + __popc(b1 & lt);
        if (isf0) { sId[2 * lane] = id0; sBody[id0] = bi; }
        if (isf1) { sId[2 * lane + 1] = id0 + isf0; sBody[id0 + isf0] = bj; }
        if (lane == 0) sCtl[3] = __popc(b0) + __popc(b1);
        __syncwarp();
        if (lane < np) {
            sPi[lane] = sId[sFirst[2 * lane]]; sPj[lane] = sId[sFirst[2 * lane + 1]];
            sGi[lane] = p.gm[bi]; sGj[lane] = p.gm[bj];
            const double rc = fmax(p.rcrit[bi], p.rcrit[bj]);
            sRc2[lane] = rc * rc; sInv[lane] = rc > 0.0 ? 1.0 / (0.9 * rc) : 0.0;
        }
        const int n0 = sCtl[3];
        const int b = lane < n0 ? sBody[lane] : 0;
#pragma unroll
        for (int c = 0; c < 3; ++c) {                                      // pad rows: a harmless body at (1, 0, 0)
            sY[c][lane] = lane < n0 ? p.x0[(size_t)c * p.ld + b] : (c == 0 ? 1.0 : 0.0);
            sY[3 + c][lane] = lane < n0 ? p.v0[(size_t)c * p.ld + b] : 0.0;
        }
    }
    __syncthreads();
    const int n = sCtl[3];
    const bool live = lane < n;
    const int me = live ? sBody[lane] : 0;
    for (int k = w; k < np; k += W) sC[k][lane] = sPi[k] == lane ? sGj[k] : sPj[k] == lane ? -sGi[k] : 0.0;
    // lanes beyond the pairs work on a pair of body 0 with itself and rc = 0: a term of exactly 0, no branch
    const int pi = lane < np ? sPi[lane] : 0, pj = lane < np ? sPj[lane] : 0;
    const double rc2 = lane < np ? sRc2[lane] : 0.0, inv = lane < np ? sInv[lane] : 0.0;
    __syncthreads();

    // ---- the Bulirsch-Stoer loop (every warp takes the same decisions from the same published numbers) ----
    const double mu = p.mu, hh = p.h, tol = p.tol;
    double t = 0.0;
    ResCtl ctl{hh, 5, 0};
    int fail = 0, nacc = 0, nrhs = 0;
    bool havef0 = false;
    double f0[3] = {0.0, 0.0, 0.0}, isx = 0.0, isv = 0.0;                  // f(y) and the inverse error scales of this body
    while (!fail) {
        const double rem = hh - t;
        if (fabs(rem) <= 4.0 * 2.220446049250313e-16 * fabs(hh)) break;
        bool last = false;
        if (fabs(ctl.H) >= fabs(rem)) { ctl.H = rem; last = true; }
        const double H = ctl.H;
        const int kcols = min(ctl.ktarg + 1, RES_KMAX - 1);
        // this warp's column: the modified midpoint rule with 2 (w + 1) substeps over H (a warp beyond the columns this
        // step tries evaluates f(y) only, when it is still missing)
        {
            const bool run = w <= kcols;
            const int nsub = 2 * (w + 1);
            const double hs = H / (double)nsub;
            double d0[6], d1[6], cur[6];
#pragma unroll
            for (int c = 0; c < 6; ++c) { d0[c] = 0.0; d1[c] = 0.0; cur[c] = 0.0; }
            if (havef0 && live) {
#pragma unroll
                for (int c = 0; c < 3; ++c) { d1[c] = hs * sY[3 + c][lane]; d1[3 + c] = hs * f0[c]; }
            }
            const int mlast = run ? nsub : 0;
#pragma unroll 1
            for (int m = havef0 ? 1 : 0; m <= mlast; ++m) {
                const bool base = m == 0;
                const double y0 = sY[0][lane], y1 = sY[1][lane], y2 = sY[2][lane];
                const double v0 = sY[3][lane] + d1[3], v1 = sY[4][lane] + d1[4], v2 = sY[5][lane] + d1[5];
                sP[w][0][lane] = base ? y0 : d1[0]; sP[w][1][lane] = base ? y1 : d1[1]; sP[w][2][lane] = base ? y2 : d1[2];
                __syncwarp();
                const double z0 = y0 + d1[0], z1 = y1 + d1[1], z2 = y2 + d1[2];            // d1 = 0 when base
                const double yk = res_rsqrt(fma(z2, z2, fma(z1, z1, z0 * z0)));
                const double wk = -mu * (yk * yk * yk);
                double a0 = wk * z0, a1 = wk * z1, a2 = wk * z2;
                {                                                          // lane = pair; straight-line code: the star's term
                    // above and this chain are independent and interleave (one warp: every instruction waits for its operands)
                    double dx = sP[w][0][pj] - sP[w][0][pi], dy = sP[w][1][pj] - sP[w][1][pi], dz = sP[w][2][pj] - sP[w][2][pi];
                    if (base) { sDy[w][0][lane] = dx; sDy[w][1][lane] = dy; sDy[w][2][lane] = dz; }
                    else { dx += sDy[w][0][lane]; dy += sDy[w][1][lane]; dz += sDy[w][2][lane]; }
                    const double u = res_pair_u_nb(fma(dz, dz, fma(dy, dy, dx * dx)), rc2, inv);
                    sFt[w][0][lane] = u * dx; sFt[w][1][lane] = u * dy; sFt[w][2][lane] = u * dz;
                }
                __syncwarp();
#pragma unroll 2
                for (int k = 0; k < np; ++k) {                             // lane = body: its terms in list order (0 for the pairs it is not in)
                    const double g = sC[k][lane];
                    a0 = fma(g, sFt[w][0][k], a0); a1 = fma(g, sFt[w][1][k], a1); a2 = fma(g, sFt[w][2][k], a2);
                }
                if (w == 0) ++nrhs;
                if (base) {                                                // f(y) and the error scales of this BS step
                    if (live) {
                        f0[0] = a0; f0[1] = a1; f0[2] = a2;
                        const double sx2 = fma(y2, y2, fma(y1, y1, y0 * y0)), sv2 = fma(v2, v2, fma(v1, v1, v0 * v0));
                        isx = sx2 > 0.0 ? res_rsqrt(sx2) : 1e300; isv = sv2 > 0.0 ? res_rsqrt(sv2) : 1e300;
                        d1[0] = hs * v0; d1[1] = hs * v1; d1[2] = hs * v2; d1[3] = hs * a0; d1[4] = hs * a1; d1[5] = hs * a2;
                    }
                    havef0 = true;
                } else if (m < nsub) {
                    const double h2s = 2.0 * hs;
                    double tt;
                    tt = fma(h2s, v0, d0[0]); d0[0] = d1[0]; d1[0] = tt;
                    tt = fma(h2s, v1, d0[1]); d0[1] = d1[1]; d1[1] = tt;
                    tt = fma(h2s, v2, d0[2]); d0[2] = d1[2]; d1[2] = tt;
                    tt = fma(h2s, a0, d0[3]); d0[3] = d1[3]; d1[3] = tt;
                    tt = fma(h2s, a1, d0[4]); d0[4] = d1[4]; d1[4] = tt;
                    tt = fma(h2s, a2, d0[5]); d0[5] = d1[5]; d1[5] = tt;
                } else {
                    cur[0] = 0.5 * (d0[0] + fma(hs, v0, d1[0])); cur[1] = 0.5 * (d0[1] + fma(hs, v1, d1[1])); cur[2] = 0.5 * (d0[2] + fma(hs, v2, d1[2]));
                    cur[3] = 0.5 * (d0[3] + fma(hs, a0, d1[3])); cur[4] = 0.5 * (d0[4] + fma(hs, a1, d1[4])); cur[5] = 0.5 * (d0[5] + fma(hs, a2, d1[5]));
                }
            }
            if (run) {
#pragma unroll
                for (int c = 0; c < 6; ++c) sCol[w][c][lane] = cur[c];
                // column w is there: warp 0, which is through with its own two substeps long before, takes the rows of
                // the tableau as the columns come in (named barrier w: this warp arrives, warp 0 waits)
                if (w > 0) { __threadfence_block(); res_nb_arrive(w, 64); }
            }
        }
        if (w == 0) {
            nrhs += (kcols + 1) * (kcols + 2) - 2;                         // the other columns' right-hand sides: sum of 2 (k + 1)
            int acc = -1, klast = 0;
            float facCur = 1.0f, facPrev = 1.0f;
            bool done = false;
#pragma unroll 1
            for (int k = 0; k <= kcols; ++k) {
                if (k > 0) res_nb_sync(k, 64);
                if (done) continue;                                        // (the later columns still have to be waited for)
                double cur[6], prev[6];
#pragma unroll
                for (int c = 0; c < 6; ++c) { cur[c] = live ? sCol[k][c][lane] : 0.0; prev[c] = cur[c]; }
                double err = 0.0;
                if (live) {
#pragma unroll 1
                    for (int j = 1; j <= k; ++j) {                         // row k of the tableau from row k-1 (in sCol[0..k-1]), overwriting it
                        const double cf = RES_COEF[k * RES_KMAX + j];
#pragma unroll
                        for (int c = 0; c < 6; ++c) {
                            const double oldv = sCol[j - 1][c][lane];
                            sCol[j - 1][c][lane] = cur[c];
                            prev[c] = cur[c];
                            cur[c] = fma(cur[c] - oldv, cf, cur[c]);
                        }
                    }
#pragma unroll
                    for (int c = 0; c < 6; ++c) {
                        sCol[k][c][lane] = cur[c];
                        double e = fabs(cur[c] - prev[c]) * (c < 3 ? isx : isv);
                        if (!(e <= 1e300)) e = 1e300;                       // NaN / inf: never accepted
                        err = fmax(err, e);
                    }
                }
                if (k >= 1) {
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) err = fmax(err, __shfl_xor_sync(full, err, o));
                    const double e = err / tol;
                    facPrev = facCur; facCur = res_fac(e, k);
                    klast = k;
                    if (e <= 1.0) { acc = k; done = true; }
                    else if (k < kcols && res_hopeless(e, k, ctl.ktarg)) done = true;
                }
            }
            if (acc >= 0 && live) {                                        // every column has read the old state by now
#pragma unroll
                for (int c = 0; c < 6; ++c) sY[c][lane] += sCol[acc][c][lane];
            }
            if (lane == 0) { sCtl[1] = acc; sCtl[2] = klast; sFac[0] = facCur; sFac[1] = facPrev; }
        }
        __syncthreads();
        const int acc = sCtl[1], klast = sCtl[2];
        const float facCur = sFac[0], facPrev = sFac[1];
        if (acc < 0) {
            if (ctl.rejected(klast, facCur)) fail = 1;
            continue;
        }
        t = last ? hh : t + H;
        ++nacc;
        havef0 = false;
        ctl.accepted(acc, facCur, facPrev);
    }
    if (w == 0) {
        if (!fail && live && (own < 0 || own == me)) {                     // a detached body's system writes only that body
#pragma unroll
            for (int c = 0; c < 3; ++c) { p.x[(size_t)c * p.ld + me] = sY[c][lane]; p.v[(size_t)c * p.ld + me] = sY[3 + c][lane]; }
        }
        if (lane == 0) {
            atomicAdd(&p.out->bodies, own < 0 ? n : 1); atomicAdd(&p.out->steps, nacc); atomicAdd(&p.out->rhs, nrhs);
            if (fail) { atomicAdd(&p.out->fail, 1); atomicAdd(&p.st->resolve_fail, 1); }
        }
    }
    }   // systems
}

// ---- class D: components of any size.  All per-body and per-pair state lives in global pools (planes of
// dbodyN / cap entries; the component's slices start at `bo` / `ps`), every phase is a thread-strided loop.  Bodies with
// more than RES_D_HUB pairs are summed by the whole block (fixed-order block_sum3), bodies with more than RES_HEAVY
// by a warp, the rest by their thread.  Slow next to the register kernels (every right-hand side streams the state
// through L1/L2), but there is no size limit besides the pools, which hold every body and every pair of the list. ----
constexpr int RES_D_HUB = 2048;

__global__ void __launch_bounds__(RES_D_THREADS) resolve_stream_kernel(ResParams p) {
    __shared__ double sRed[32];
    __shared__ double sSum[32][3];
    __shared__ int sScan[64];
    __shared__ int sBc[4];
    __shared__ int sHub[RES_D_HMAX];
    __shared__ double sHubAcc[RES_D_HMAX][3];
    constexpr int NT = RES_D_THREADS;
    constexpr unsigned full = 0xffffffffu;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid < 64) sScan[tid] = 0;
    const long long cap = p.cap, BN = p.dbodyN;
    const int npAll = (int)p.st->nce_last;

    for (;;) {
    __syncthreads();
    if (tid == 0) sBc[0] = atomicAdd(&p.ctl[RES_CTL_TKT + 4], 1);
    __syncthreads();
    const int ticket = sBc[0];
    if (ticket >= p.ctl[RES_CTL_CNT + 4]) break;
    const int comp = p.clist[(size_t)4 * cap + ticket];
    const int np = p.cnp[comp];
    const int ps = p.cstart[comp];
    double* const F = p.dpair + ps;                       // planes 0..2: pair terms; 3 rc2, 4 inv, 5 gm_i, 6 gm_j
    int* const Qs = p.dpairi + ps;                        // plane 0: the component's pairs in list order; 1, 2: global members;
    int* const Bi = Qs + cap; int* const Bj = Bi + cap;   // 3, 4: local members; 5: second-member adjacency
    int* const Pi = Bj + cap; int* const Pj = Pi + cap; int* const Adj = Pj + cap; int* const Adj2 = Adj + cap;
    const int ownb = res_owner(p, p.cq[ps], p.label);       // the component's smallest body
    const int own = p.cown[comp];
    if (own >= 0) {                                         // a detached body whose partners' components grew past 1023 pairs after it was
        if (tid == 0) { atomicAdd(&p.out->fail, 1); atomicAdd(&p.st->resolve_fail, 1); }      // detached: not handled (reported)
        continue;
    }

    // ---- pairs in list order: stable compaction of the whole list ----
    {
        int cnt = 0;
        for (int base = 0; base < npAll; base += NT) {
            const int q = base + tid;
            const int mine = (q < npAll && res_owner(p, q, p.label) == ownb) ? 1 : 0;
            int tot;
            const int off = res_scan(mine, sScan, tot);
            if (mine) Qs[cnt + off] = q;
            cnt += tot;
        }
    }
    __syncthreads();
    for (int k = tid; k < np; k += NT) {
        const int q = Qs[k], bi = p.pairs[2 * q], bj = p.pairs[2 * q + 1];
        Bi[k] = bi; Bj[k] = bj;
        p.loc[bi] = 0x7fffffff; p.loc[bj] = 0x7fffffff;
    }
    __syncthreads();
    for (int k = tid; k < np; k += NT) { atomicMin(&p.loc[Bi[k]], 2 * k); atomicMin(&p.loc[Bj[k]], 2 * k + 1); }
    __syncthreads();
    int n = 0;
    for (int base = 0; base < np; base += NT) {           // count the bodies, then take a slice of the body pool
        const int k = base + tid;
        int f = 0;
        if (k < np) f = ((p.loc[Bi[k]] == 2 * k) ? 1 : 0) + ((p.loc[Bj[k]] == 2 * k + 1) ? 1 : 0);
        int tot;
        res_scan(f, sScan, tot);
        n += tot;
    }
    if (tid == 0) sBc[1] = atomicAdd(&p.ctl[RES_CTL_POOL], n);
    __syncthreads();
    const long long bo = sBc[1];
    if (bo + n > BN) {                                    // cannot happen while the pool holds every listed body
        if (tid == 0) { atomicAdd(&p.out->fail, 1); atomicAdd(&p.st->resolve_fail, 1); atomicAdd(&p.out->bodies, n); }
        continue;
    }
    double* const B = p.dbody + bo;                       // double planes: see RES_D_BODY_PLANES
    int* const Body = p.dbodyi + bo;                      // int planes: body, iLo, iHi, jLo, d2
    int* const ILo = Body + BN; int* const IHi = ILo + BN; int* const JLo = IHi + BN; int* const D2 = JLo + BN;
    int* const Tier = D2 + BN; int* const WList = Tier + BN;   // tier: 0 summed by its thread, 1 by a warp, 2 + h by the block (hub h)
    {
        int cnt = 0;
        for (int base = 0; base < np; base += NT) {
            const int k = base + tid;
            int fi = 0, fj = 0;
            if (k < np) { fi = (p.loc[Bi[k]] == 2 * k) ? 1 : 0; fj = (p.loc[Bj[k]] == 2 * k + 1) ? 1 : 0; }
            int tot;
            const int off = res_scan(fi + fj, sScan, tot);
            if (fi) Body[cnt + off] = Bi[k];
            if (fj) Body[cnt + off + fi] = Bj[k];
            cnt += tot;
        }
    }
    __syncthreads();
    for (int id = tid; id < n; id += NT) { p.loc[Body[id]] = id; ILo[id] = 0; IHi[id] = 0; D2[id] = 0; }
    __syncthreads();
    for (int k = tid; k < np; k += NT) {
        const int bi = Bi[k], bj = Bj[k];
        const int li = p.loc[bi], lj = p.loc[bj];
        Pi[k] = li; Pj[k] = lj;
        F[5 * cap + k] = p.gm[bi]; F[6 * cap + k] = p.gm[bj];
        const double rc = fmax(p.rcrit[bi], p.rcrit[bj]);
        F[3 * cap + k] = rc * rc; F[4 * cap + k] = rc > 0.0 ? 1.0 / (0.9 * rc) : 0.0;
        if (k == 0 || Bi[k - 1] != bi) ILo[li] = k;
        if (k == np - 1 || Bi[k + 1] != bi) IHi[li] = k + 1;
        atomicAdd(&D2[lj], 1);
    }
    __syncthreads();
    {
        int carry = 0;
        for (int base = 0; base < n; base += NT) {
            const int id = base + tid;
            int tot;
            const int off = res_scan(id < n ? D2[id] : 0, sScan, tot);
            if (id < n) JLo[id] = carry + off;
            carry += tot;
        }
    }
    __syncthreads();
    // second-member lists in list order: slots taken in arrival order (Tier = fill counter for now), then every list
    // of more than one entry rank-sorted by a warp (sum of d2^2 / 32 steps instead of np^2 / NT)
    for (int id = tid; id < n; id += NT) Tier[id] = 0;
    __syncthreads();
    for (int k = tid; k < np; k += NT) { const int lj = Pj[k]; Adj2[JLo[lj] + atomicAdd(&Tier[lj], 1)] = k; }
    __syncthreads();
    for (int id = warp; id < n; id += NT / 32) {
        const int j0 = JLo[id], dj = D2[id];
        for (int e = lane; e < dj; e += 32) {
            const int mine = Adj2[j0 + e];
            int r = 0;
            for (int m = 0; m < dj; ++m) r += (Adj2[j0 + m] < mine) ? 1 : 0;
            Adj[j0 + r] = mine;
        }
    }
    __syncthreads();
    // hubs (block-summed) and warp-summed bodies, in body order
    int nhub = 0, nwl = 0;
    for (int base = 0; base < n; base += NT) {
        const int id = base + tid;
        const int deg = id < n ? D2[id] + IHi[id] - ILo[id] : 0;
        int totH, totW;
        const int hubIdx = nhub + res_scan(deg > RES_D_HUB ? 1 : 0, sScan, totH);
        const bool isHub = deg > RES_D_HUB && hubIdx < RES_D_HMAX;
        if (isHub) sHub[hubIdx] = id;
        nhub += totH;
        const bool isW = deg > RES_HEAVY && !isHub;
        const int offW = res_scan(isW ? 1 : 0, sScan, totW);
        if (isW) WList[nwl + offW] = id;
        nwl += totW;
        if (id < n) Tier[id] = isHub ? 2 + hubIdx : isW ? 1 : 0;
    }
    if (nhub > RES_D_HMAX) nhub = RES_D_HMAX;
    __syncthreads();
    for (int id = tid; id < n; id += NT) {
        const int b = Body[id];
#pragma unroll
        for (int c = 0; c < 3; ++c) { B[(3 + c) * BN + id] = p.x0[(size_t)c * p.ld + b]; B[(6 + c) * BN + id] = p.v0[(size_t)c * p.ld + b]; }
    }
    __syncthreads();

    const double mu = p.mu, hh = p.h, tol = p.tol;
    int nrhs = 0;
    // a(P) -> ACC planes (26..28).  src: 0 positions = Y (P holds Y), 1 positions = Y + D1 (P holds the increments D1)
    auto accel = [&](int src) {
        for (int id = tid; id < n; id += NT) {
#pragma unroll
            for (int c = 0; c < 3; ++c) B[c * BN + id] = src ? B[(15 + c) * BN + id] : B[(3 + c) * BN + id];
        }
        __syncthreads();
        for (int k = tid; k < np; k += NT) {
            const int i = Pi[k], j = Pj[k];
            double dx = B[j] - B[i], dy = B[BN + j] - B[BN + i], dz = B[2 * BN + j] - B[2 * BN + i];
            if (src) { dx += F[7 * cap + k]; dy += F[8 * cap + k]; dz += F[9 * cap + k]; }      // (y_j - y_i) + (dl_j - dl_i), see rhs above
            else { F[7 * cap + k] = dx; F[8 * cap + k] = dy; F[9 * cap + k] = dz; }
            const double u = res_pair_u(fma(dz, dz, fma(dy, dy, dx * dx)), F[3 * cap + k], F[4 * cap + k]);
            F[k] = u * dx; F[cap + k] = u * dy; F[2 * cap + k] = u * dz;
        }
        __syncthreads();
        for (int hI = 0; hI < nhub; ++hI) {
            const int id = sHub[hI];
            const int j0 = JLo[id], dj = D2[id], i0 = ILo[id], i1 = IHi[id];
            double h0 = 0.0, h1 = 0.0, h2 = 0.0;
            for (int e = tid; e < dj; e += NT) {
                const int k = Adj[j0 + e];
                const double g = F[5 * cap + k];
                h0 = fma(-g, F[k], h0); h1 = fma(-g, F[cap + k], h1); h2 = fma(-g, F[2 * cap + k], h2);
            }
            for (int k = i0 + tid; k < i1; k += NT) {
                const double g = F[6 * cap + k];
                h0 = fma(g, F[k], h0); h1 = fma(g, F[cap + k], h1); h2 = fma(g, F[2 * cap + k], h2);
            }
            __syncthreads();                              // sSum free
            block_sum3<NT>(h0, h1, h2, sSum);
            if (tid == 0) { sHubAcc[hI][0] = h0; sHubAcc[hI][1] = h1; sHubAcc[hI][2] = h2; }
        }
        // bodies summed by a warp, dealt round-robin
        for (int wi = warp; wi < nwl; wi += NT / 32) {
            const int id = WList[wi];
            const int dj = D2[id], i0 = ILo[id], i1 = IHi[id];
            const int j0 = JLo[id];
            double h0 = 0.0, h1 = 0.0, h2 = 0.0;
            for (int e = lane; e < dj; e += 32) {
                const int k = Adj[j0 + e];
                const double g = F[5 * cap + k];
                h0 = fma(-g, F[k], h0); h1 = fma(-g, F[cap + k], h1); h2 = fma(-g, F[2 * cap + k], h2);
            }
            for (int k = i0 + lane; k < i1; k += 32) {
                const double g = F[6 * cap + k];
                h0 = fma(g, F[k], h0); h1 = fma(g, F[cap + k], h1); h2 = fma(g, F[2 * cap + k], h2);
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                h0 += __shfl_xor_sync(full, h0, o); h1 += __shfl_xor_sync(full, h1, o); h2 += __shfl_xor_sync(full, h2, o);
            }
            if (lane == 0) { B[26 * BN + id] = h0; B[27 * BN + id] = h1; B[28 * BN + id] = h2; }
        }
        __syncthreads();
        for (int id = tid; id < n; id += NT) {
            double z0 = B[id], z1 = B[BN + id], z2 = B[2 * BN + id];
            if (src) { z0 += B[3 * BN + id]; z1 += B[4 * BN + id]; z2 += B[5 * BN + id]; }
            const double yk = res_rsqrt(fma(z2, z2, fma(z1, z1, z0 * z0)));
            const double w = -mu * (yk * yk * yk);
            double a0 = w * z0, a1 = w * z1, a2 = w * z2;
            const int tier = Tier[id];
            if (tier >= 2) { a0 += sHubAcc[tier - 2][0]; a1 += sHubAcc[tier - 2][1]; a2 += sHubAcc[tier - 2][2]; }
            else if (tier == 1) { a0 += B[26 * BN + id]; a1 += B[27 * BN + id]; a2 += B[28 * BN + id]; }
            else {
                const int dj = D2[id], i0 = ILo[id], i1 = IHi[id], j0 = JLo[id];
                for (int e = 0; e < dj; ++e) { const int k = Adj[j0 + e]; const double g = F[5 * cap + k]; a0 = fma(-g, F[k], a0); a1 = fma(-g, F[cap + k], a1); a2 = fma(-g, F[2 * cap + k], a2); }
                for (int k = i0; k < i1; ++k) { const double g = F[6 * cap + k]; a0 = fma(g, F[k], a0); a1 = fma(g, F[cap + k], a1); a2 = fma(g, F[2 * cap + k], a2); }
            }
            B[26 * BN + id] = a0; B[27 * BN + id] = a1; B[28 * BN + id] = a2;
        }
        ++nrhs;
        // every thread reads back only the accelerations it wrote: no barrier needed here
    };

    double t = 0.0;
    ResCtl ctl{hh, 5, 0};
    int fail = 0, nacc = 0;
    bool havef0 = false;
    while (!fail) {
        const double rem = hh - t;
        if (fabs(rem) <= 4.0 * 2.220446049250313e-16 * fabs(hh)) break;
        bool last = false;
        if (fabs(ctl.H) >= fabs(rem)) { ctl.H = rem; last = true; }
        const double H = ctl.H;
        if (!havef0) {
            accel(0);
            for (int id = tid; id < n; id += NT) {
                double s2x = 0.0, s2v = 0.0;
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    B[(21 + c) * BN + id] = B[(26 + c) * BN + id];
                    const double xx = B[(3 + c) * BN + id], vv = B[(6 + c) * BN + id];
                    s2x = fma(xx, xx, s2x); s2v = fma(vv, vv, s2v);
                }
                B[24 * BN + id] = sqrt(s2x); B[25 * BN + id] = sqrt(s2v);
            }
            havef0 = true;
        }
        const int kcols = min(ctl.ktarg + 1, RES_KMAX - 1);
        int acc = -1, klast = 0;
        float facCur = 1.0f, facPrev = 1.0f;
        for (int k = 0; k <= kcols; ++k) {
            const int nsub = 2 * (k + 1);
            const double hs = H / (double)nsub;
            for (int id = tid; id < n; id += NT) {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    B[(9 + c) * BN + id] = 0.0; B[(12 + c) * BN + id] = 0.0;
                    B[(15 + c) * BN + id] = hs * B[(6 + c) * BN + id]; B[(18 + c) * BN + id] = hs * B[(21 + c) * BN + id];
                }
            }
            double err = 0.0;
            for (int m = 1; m <= nsub; ++m) {
                accel(1);
                for (int id = tid; id < n; id += NT) {
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        const double d0x = B[(9 + c) * BN + id], d0v = B[(12 + c) * BN + id];
                        const double d1x = B[(15 + c) * BN + id], d1v = B[(18 + c) * BN + id];
                        const double fx = B[(6 + c) * BN + id] + d1v, fv = B[(26 + c) * BN + id];
                        if (m < nsub) {
                            B[(9 + c) * BN + id] = d1x; B[(12 + c) * BN + id] = d1v;
                            B[(15 + c) * BN + id] = fma(2.0 * hs, fx, d0x); B[(18 + c) * BN + id] = fma(2.0 * hs, fv, d0v);
                        } else {
                            const double r2[2] = {0.5 * (d0x + fma(hs, fx, d1x)), 0.5 * (d0v + fma(hs, fv, d1v))};
#pragma unroll
                            for (int hv = 0; hv < 2; ++hv) {          // position component c, then velocity component c
                                double* Tb = B + (size_t)(29 + hv * 3 + c) * BN + id;      // T_{., j} at plane 29 + j*6 + comp
                                double cur = r2[hv], prev = 0.0;
                                for (int j = 1; j <= k; ++j) {
                                    const double oldv = Tb[(size_t)(j - 1) * 6 * BN];
                                    Tb[(size_t)(j - 1) * 6 * BN] = cur;
                                    prev = cur;
                                    cur = fma(cur - oldv, RES_COEF[k * RES_KMAX + j], cur);
                                }
                                Tb[(size_t)k * 6 * BN] = cur;
                                if (k >= 1) {
                                    double e = fabs(cur - prev);
                                    const double sc = B[(24 + hv) * BN + id];
                                    e = sc > 0.0 ? e / sc : (e > 0.0 ? 1e300 : 0.0);
                                    if (!(e <= 1e300)) e = 1e300;
                                    err = fmax(err, e);
                                }
                            }
                        }
                    }
                }
            }
            if (k >= 1) {
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) err = fmax(err, __shfl_xor_sync(full, err, o));
                __syncthreads();
                if (lane == 0) sRed[warp] = err;
                __syncthreads();
                double e = sRed[0];
#pragma unroll
                for (int w = 1; w < NT / 32; ++w) e = fmax(e, sRed[w]);
                e /= tol;
                facPrev = facCur; facCur = res_fac(e, k);
                klast = k;
                if (e <= 1.0) { acc = k; break; }
                if (k < kcols && res_hopeless(e, k, ctl.ktarg)) break;
            }
        }
        if (acc < 0) {
            if (ctl.rejected(klast, facCur)) fail = 1;
            continue;
        }
        for (int id = tid; id < n; id += NT) {
#pragma unroll
            for (int c = 0; c < 6; ++c) B[(3 + c) * BN + id] += B[(size_t)(29 + acc * 6 + c) * BN + id];
        }
        t = last ? hh : t + H;
        ++nacc;
        havef0 = false;
        ctl.accepted(acc, facCur, facPrev);
    }
    if (!fail) {
        for (int id = tid; id < n; id += NT) {
            const int b = Body[id];
            if (own >= 0 && own != b) continue;
#pragma unroll
            for (int c = 0; c < 3; ++c) { p.x[(size_t)c * p.ld + b] = B[(3 + c) * BN + id]; p.v[(size_t)c * p.ld + b] = B[(6 + c) * BN + id]; }
        }
    }
    if (tid == 0) {
        atomicAdd(&p.out->bodies, own < 0 ? n : 1); atomicAdd(&p.out->steps, nacc); atomicAdd(&p.out->rhs, nrhs);
        if (fail) { atomicAdd(&p.out->fail, 1); atomicAdd(&p.st->resolve_fail, 1); }
    }
    }   // components
}

}  // namespace mopal
