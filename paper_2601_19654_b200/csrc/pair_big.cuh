// pair_big.cuh - the big x all pair sum for few gravity sources (the paper's own loop bounds
// `do j = 2, nbod` x `do i = 2, nbig`, with N_big <= ~100 and N_small up to
// 1e6):  a_i = sum_{j < nbig, j != i} gm_j K_ij (x_j - x_i) / r_ij^3  for EVERY i.
//
// With so few sources there is nothing to split and nothing to stream: a persistent grid (a few
// CTAs per SM) walks over blocks of bodies i; each CTA stages the source records {x, y, z, gm} in
// shared memory (once if nbig <= BIG_SRC, else BIG_SRC at a time), every thread keeps IPT
// bodies i in registers (the next block's prefetched), sweeps the sources in ascending j (fixed order, one accumulator per
// component - bit-reproducible) and writes a_i itself, with the closing half kick
// v += hk a (Hamiltonian block LOOP 1) fused in.  No partial buffers, no
// reduce kernel.  The per-pair arithmetic is pair_accel_kernel's (16 FP64-pipe instructions
// on the K = 1 path, integer gate on the high word of s2), except that the gate is per source,
// not per tile - a giant's rcrit (1-2 AU) must not send every pair of the staged sources down
// the changeover path - and that path is in line (changeover_weight).
#pragma once
#include "common.cuh"
#include "pair_accel.cuh"

namespace mopal {

constexpr int BIG_THREADS = 128;
constexpr int BIG_SRC = 1024;        // sources staged per pass (32 KB of shared memory)

struct BigParams {
    const double* x;       // 3*ld, positions (after the jump)
    const double* gm;      // nb
    const double* rcrit;   // nb
    double* a;             // 3*ld out
    double* v;             // 3*ld in/out when KICK
    int nb, nbig, ld;
    double hk;
    int blk0, blk1;        // pair_big_kernel: the blocks of bodies i this launch covers (a rank's share, row f4), blk1 <= 0: all
};

// The pairs the integer gate could not prove to be outside the changeover shell (readings A-1..A-5,
// A-9): w = gm_j / r^3 from the fast path (already exact to rounding) times K(r; rc).  In line and
// on registers / shared memory only - with a giant among the sources some lane of most warps is
// inside its shell, so this path is not rare per warp.
__device__ __forceinline__ double changeover_weight(double s2, double w, double rc) {
    if (!(s2 > 0.0)) return 0.0;              // self pair, coincident bodies (w is NaN there)
    const double rc2 = rc * rc;
    if (s2 >= rc2) return w;                  // K = 1 (the gate compares high words only)
    const double rin = 0.1 * rc;
    if (s2 <= rin * rin) return 0.0;          // K = 0
    const double q = (sqrt(s2) - rin) / (0.9 * rc);
    return w * (q * q * q * (10.0 + q * (6.0 * q - 15.0)));
}

template <int IPT, int U, bool KICK>
__global__ void __launch_bounds__(BIG_THREADS) pair_big_kernel(BigParams p) {
    __shared__ __align__(16) double2 s_src[2 * BIG_SRC];
    __shared__ int s_gj[BIG_SRC];      // per-source changeover gate: high word of rcrit_j^2
    __shared__ double s_rc[BIG_SRC];   // rcrit_j, for the pairs that fail the gate
    const int tid = threadIdx.x;
    const int nIall = (p.nb + BIG_THREADS * IPT - 1) / (BIG_THREADS * IPT);
    const int nIblk = p.blk1 > 0 ? min(p.blk1, nIall) : nIall;
    const int blkFirst = p.blk1 > 0 ? p.blk0 : 0;
    const bool single = p.nbig <= BIG_SRC;             // all sources fit: staged once per CTA

    auto stage = [&](int j0, int n, int npad) {
        for (int t = tid; t < npad; t += BIG_THREADS) {
            const int j = j0 + t;
            if (t < n) {
                s_src[2 * t] = make_double2(p.x[j], p.x[p.ld + j]);
                s_src[2 * t + 1] = make_double2(p.x[2 * p.ld + j], p.gm[j]);
                const double rc = p.rcrit[j];
                s_gj[t] = __double2hiint(rc * rc);
                s_rc[t] = rc;
            } else {                                   // far away and massless: contributes exactly 0
                s_src[2 * t] = make_double2(PAD_POS, PAD_POS);
                s_src[2 * t + 1] = make_double2(PAD_POS, 0.0);
                s_gj[t] = 0;
                s_rc[t] = 0.0;
            }
        }
    };
    if (single) {
        stage(0, p.nbig, (p.nbig + U - 1) / U * U);
        __syncthreads();
    }

    // the CTA walks over blocks of BIG_THREADS * IPT bodies i; the next block's bodies are loaded
    // while the current block is summed
    double nx[IPT], ny[IPT], nz[IPT], nrc[IPT];
    auto fetch = [&](int blk) {
#pragma unroll
        for (int k = 0; k < IPT; ++k) {
            const int i = blk * (BIG_THREADS * IPT) + tid + k * BIG_THREADS;
            const bool ok = blk < nIblk && i < p.nb;
            nx[k] = ok ? p.x[i] : 0.0; ny[k] = ok ? p.x[p.ld + i] : 0.0; nz[k] = ok ? p.x[2 * p.ld + i] : 0.0;
            nrc[k] = ok ? p.rcrit[i] : 0.0;
        }
    };
    fetch(blkFirst + blockIdx.x);
    for (int blk = blkFirst + blockIdx.x; blk < nIblk; blk += gridDim.x) {
        const int ibase = blk * (BIG_THREADS * IPT) + tid;
        double xi[IPT], yi[IPT], zi[IPT], ax[IPT], ay[IPT], az[IPT], rci[IPT];
        int gi[IPT];
#pragma unroll
        for (int k = 0; k < IPT; ++k) {
            xi[k] = nx[k]; yi[k] = ny[k]; zi[k] = nz[k]; rci[k] = nrc[k];
            gi[k] = __double2hiint(rci[k] * rci[k]);
            ax[k] = ay[k] = az[k] = 0.0;
        }
        fetch(blk + gridDim.x);
        // the velocities the closing kick updates: loaded now, needed after the sweep
        double vx[IPT], vy[IPT], vz[IPT];
        if (KICK) {
#pragma unroll
            for (int k = 0; k < IPT; ++k) {
                const int i = ibase + k * BIG_THREADS;
                const bool ok = i < p.nb;
                vx[k] = ok ? p.v[i] : 0.0; vy[k] = ok ? p.v[p.ld + i] : 0.0; vz[k] = ok ? p.v[2 * p.ld + i] : 0.0;
            }
        }

        for (int j0 = 0; j0 < p.nbig; j0 += BIG_SRC) {
            const int n = min(BIG_SRC, p.nbig - j0);
            const int npad = (n + U - 1) / U * U;
            if (!single) {
                __syncthreads();                       // previous chunk fully consumed
                stage(j0, n, npad);
                __syncthreads();
            }
            // the records of the next U sources are read from shared memory while the current ones are used
            double2 qa[U], qb[U];
            int qg[U];
#pragma unroll
            for (int u = 0; u < U; ++u) { qa[u] = s_src[2 * u]; qb[u] = s_src[2 * u + 1]; qg[u] = s_gj[u]; }
#pragma unroll 1
            for (int jj = 0; jj < npad; jj += U) {
                double dx[U][IPT], dy[U][IPT], dz[U][IPT], w[U][IPT];
                bool any = false;
                double2 ca[U], cb[U];
                int cg[U];
                const int jn = min(jj + U, npad - U);            // last pass re-reads its own records
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    ca[u] = qa[u]; cb[u] = qb[u]; cg[u] = qg[u];
                    qa[u] = s_src[2 * (jn + u)]; qb[u] = s_src[2 * (jn + u) + 1]; qg[u] = s_gj[jn + u];
                }
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    const double2 pa = ca[u];      // x, y
                    const double2 pb = cb[u];      // z, gm
                    const int gj = cg[u];
#pragma unroll
                    for (int k = 0; k < IPT; ++k) {
                        const double ddx = pa.x - xi[k], ddy = pa.y - yi[k], ddz = pb.x - zi[k];
                        const double s2 = fma(ddz, ddz, fma(ddy, ddy, ddx * ddx));
                        const double y = rsqrt_seed(s2);
                        const double y2 = y * y;
                        const double e = fma(-s2, y2, 1.0);
                        const double w0 = (pb.y * y) * y2;
                        const double t = e * fma(1.875, e, 1.5);
                        w[u][k] = fma(w0, t, w0);
                        any |= (__double2hiint(s2) <= max(gi[k], gj));
                        dx[u][k] = ddx; dy[u][k] = ddy; dz[u][k] = ddz;
                    }
                }
                if (any) {  // changeover shell, self pair, coincident bodies
#pragma unroll
                    for (int u = 0; u < U; ++u) {
#pragma unroll
                        for (int k = 0; k < IPT; ++k) {
                            const double s2 = fma(dz[u][k], dz[u][k], fma(dy[u][k], dy[u][k], dx[u][k] * dx[u][k]));
                            if (__double2hiint(s2) <= max(gi[k], s_gj[jj + u]))
                                w[u][k] = changeover_weight(s2, w[u][k], fmax(rci[k], s_rc[jj + u]));
                        }
                    }
                }
#pragma unroll
                for (int u = 0; u < U; ++u) {
#pragma unroll
                    for (int k = 0; k < IPT; ++k) {
                        ax[k] = fma(w[u][k], dx[u][k], ax[k]);
                        ay[k] = fma(w[u][k], dy[u][k], ay[k]);
                        az[k] = fma(w[u][k], dz[u][k], az[k]);
                    }
                }
            }
        }

#pragma unroll
        for (int k = 0; k < IPT; ++k) {
            const int i = ibase + k * BIG_THREADS;
            if (i < p.nb) {
                p.a[i] = ax[k]; p.a[p.ld + i] = ay[k]; p.a[2 * p.ld + i] = az[k];
                if (KICK) {
                    p.v[i] = fma(p.hk, ax[k], vx[k]);
                    p.v[p.ld + i] = fma(p.hk, ay[k], vy[k]);
                    p.v[2 * p.ld + i] = fma(p.hk, az[k], vz[k]);
                }
            }
        }
    }
}

// ---- small systems (nb <= PSM_MAX; the paper's own regime is N <= 1000) -------------
// There are too few bodies to fill the chip with one thread per body, so G lanes share a body: lane g
// sums the sources j = g, g + G, ... of each staged chunk (ascending), the G partial sums are combined by a
// fixed shuffle tree, lane 0 writes a_i (and the closing kick).  Sources are staged in shared memory; same per-pair
// arithmetic, per-source gate and in-line changeover weight as pair_big_kernel.  One launch replaces
// pack + pair + reduce.
constexpr int PSM_MAX = 8191;         // above: the two-sided kernel
constexpr int PSM_CHUNK = 1024;       // sources staged per pass
constexpr int PSM_THREADS = 128;

template <int G, bool KICK>
__global__ void __launch_bounds__(PSM_THREADS) pair_small_kernel(BigParams p) {
    __shared__ __align__(16) double2 s_src[2 * PSM_CHUNK];
    __shared__ int s_gj[PSM_CHUNK];
    __shared__ double s_rc[PSM_CHUNK];
    const int tid = threadIdx.x;
    const int i = blockIdx.x * (PSM_THREADS / G) + tid / G;
    const int g = tid % G;
    const bool live = i < p.nb;
    const double xi = live ? p.x[i] : 0.0, yi = live ? p.x[p.ld + i] : 0.0, zi = live ? p.x[2 * p.ld + i] : 0.0;
    const double rci = live ? p.rcrit[i] : 0.0;
    const int gi = __double2hiint(rci * rci);
    double vx = 0.0, vy = 0.0, vz = 0.0;
    if (KICK && live && g == 0) { vx = p.v[i]; vy = p.v[p.ld + i]; vz = p.v[2 * p.ld + i]; }
    double ax = 0.0, ay = 0.0, az = 0.0;
    for (int j0 = 0; j0 < p.nbig; j0 += PSM_CHUNK) {
        const int n = min(PSM_CHUNK, p.nbig - j0);
        __syncthreads();                                   // previous chunk fully consumed
        for (int t = tid; t < n; t += PSM_THREADS) {
            const int j = j0 + t;
            s_src[2 * t] = make_double2(p.x[j], p.x[p.ld + j]);
            s_src[2 * t + 1] = make_double2(p.x[2 * p.ld + j], p.gm[j]);
            const double rc = p.rcrit[j];
            s_gj[t] = __double2hiint(rc * rc);
            s_rc[t] = rc;
        }
        __syncthreads();
#pragma unroll 4
        for (int j = g; j < n; j += G) {
            const double2 pa = s_src[2 * j], pb = s_src[2 * j + 1];
            const double dx = pa.x - xi, dy = pa.y - yi, dz = pb.x - zi;
            const double s2 = fma(dz, dz, fma(dy, dy, dx * dx));
            const double y = rsqrt_seed(s2);
            const double y2 = y * y;
            const double e = fma(-s2, y2, 1.0);
            const double w0 = (pb.y * y) * y2;
            const double t = e * fma(1.875, e, 1.5);
            double w = fma(w0, t, w0);
            if (__double2hiint(s2) <= max(gi, s_gj[j])) w = changeover_weight(s2, w, fmax(rci, s_rc[j]));
            ax = fma(w, dx, ax); ay = fma(w, dy, ay); az = fma(w, dz, az);
        }
    }
#pragma unroll
    for (int o = G / 2; o > 0; o >>= 1) {
        ax += __shfl_down_sync(0xffffffffu, ax, o, G);
        ay += __shfl_down_sync(0xffffffffu, ay, o, G);
        az += __shfl_down_sync(0xffffffffu, az, o, G);
    }
    if (live && g == 0) {
        p.a[i] = ax; p.a[p.ld + i] = ay; p.a[2 * p.ld + i] = az;
        if (KICK) {
            p.v[i] = fma(p.hk, ax, vx); p.v[p.ld + i] = fma(p.hk, ay, vy); p.v[2 * p.ld + i] = fma(p.hk, az, vz);
        }
    }
}

}  // namespace mopal
