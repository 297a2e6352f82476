// pair_big.cuh - the big x all pair sum for few gravity sources (the paper's own loop bounds
// `do j = 2, nbod` x `do i = 2, nbig`, with N_big <= ~100 and N_small up to
// 1e6):  a_i = sum_{j < nbig, j != i} gm_j K_ij (x_j - x_i) / r_ij^3  for EVERY i.
//
// With so few sources there is nothing to split and nothing to stream: each CTA stages the
// source records {x, y, z, gm} in shared memory (BIG_SRC at a time), every thread keeps IPT
// bodies i in registers, sweeps the sources in ascending j (fixed order, one accumulator per
// component - bit-reproducible) and writes a_i itself, with the closing half kick
// v += hk a (Hamiltonian block LOOP 1) fused in.  No partial buffers, no
// reduce kernel.  The per-pair arithmetic is pair_accel_kernel's (16 FP64-pipe instructions
// on the K = 1 path, integer gate on the high word of s2, slow_weight for the rest), except that
// the gate is per source, not per tile: a giant's rcrit (1-2 AU) must not send every pair of
// the staged sources down the slow path.
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
};

template <int IPT, int U, bool KICK>
__global__ void __launch_bounds__(BIG_THREADS) pair_big_kernel(BigParams p) {
    __shared__ __align__(16) double2 s_src[2 * BIG_SRC];
    __shared__ int s_gj[BIG_SRC];      // per-source changeover gate: high word of rcrit_j^2
    const int tid = threadIdx.x;
    const int ibase = blockIdx.x * (BIG_THREADS * IPT) + tid;
    double xi[IPT], yi[IPT], zi[IPT], ax[IPT], ay[IPT], az[IPT];
    int gi[IPT];
#pragma unroll
    for (int k = 0; k < IPT; ++k) {
        const int i = ibase + k * BIG_THREADS;
        if (i < p.nb) {
            xi[k] = p.x[i]; yi[k] = p.x[p.ld + i]; zi[k] = p.x[2 * p.ld + i];
            const double rc = p.rcrit[i];
            gi[k] = __double2hiint(rc * rc);
        } else {
            xi[k] = yi[k] = zi[k] = 0.0; gi[k] = 0;
        }
        ax[k] = ay[k] = az[k] = 0.0;
    }

    for (int j0 = 0; j0 < p.nbig; j0 += BIG_SRC) {
        const int n = min(BIG_SRC, p.nbig - j0);
        const int npad = (n + U - 1) / U * U;
        __syncthreads();                               // previous chunk fully consumed
        for (int t = tid; t < npad; t += BIG_THREADS) {
            const int j = j0 + t;
            if (t < n) {
                s_src[2 * t] = make_double2(p.x[j], p.x[p.ld + j]);
                s_src[2 * t + 1] = make_double2(p.x[2 * p.ld + j], p.gm[j]);
                const double rc = p.rcrit[j];
                s_gj[t] = __double2hiint(rc * rc);
            } else {                                   // far away and massless: contributes exactly 0
                s_src[2 * t] = make_double2(PAD_POS, PAD_POS);
                s_src[2 * t + 1] = make_double2(PAD_POS, 0.0);
                s_gj[t] = 0;
            }
        }
        __syncthreads();

#pragma unroll 1
        for (int jj = 0; jj < npad; jj += U) {
            double dx[U][IPT], dy[U][IPT], dz[U][IPT], w[U][IPT];
            bool any = false;
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const double2 pa = s_src[2 * (jj + u)];      // x, y
                const double2 pb = s_src[2 * (jj + u) + 1];  // z, gm
                const int gj = s_gj[jj + u];
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
            if (any) {  // rare: changeover shell, self pair, coincident bodies
#pragma unroll
                for (int u = 0; u < U; ++u) {
#pragma unroll
                    for (int k = 0; k < IPT; ++k) {
                        const double s2 = fma(dz[u][k], dz[u][k], fma(dy[u][k], dy[u][k], dx[u][k] * dx[u][k]));
                        if (__double2hiint(s2) <= max(gi[k], s_gj[jj + u]))
                            w[u][k] = (jj + u < n) ? slow_weight(s2, s_src[2 * (jj + u) + 1].y, p.rcrit,
                                                                 ibase + k * BIG_THREADS, j0 + jj + u, p.nb)
                                                   : 0.0;
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
                p.v[i] = fma(p.hk, ax[k], p.v[i]);
                p.v[p.ld + i] = fma(p.hk, ay[k], p.v[p.ld + i]);
                p.v[2 * p.ld + i] = fma(p.hk, az[k], p.v[2 * p.ld + i]);
            }
        }
    }
}

}  // namespace mopal
