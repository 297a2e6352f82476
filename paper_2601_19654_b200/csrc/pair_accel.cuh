// pair_accel.cuh - the O(N^2) K(r)-weighted mutual-gravity sum (force block LOOP 2,
// PAPER.md:150-165):  a_i = sum_{j != i} gm_j K_ij (x_j - x_i) / r_ij^3.
//
// i-parallel: every compute thread owns IPT bodies i in registers and sweeps a
// range of j-tiles that one producer warp streams into shared memory with TMA
// 1-D bulk copies (cp.async.bulk + mbarrier ring).  A tile is TJ packed records
// {x, y, z, gm} plus a 16-byte header holding the tile's changeover gate.
//
// Fast path (K = 1, all but ~1e-4 of the pairs): 16 FP64-pipe instructions,
//   3 DADD (d), DMUL + 2 DFMA (s2), MUFU.RSQ64H seed y ~ s2^-1/2 (2^-22),
//   y2 = y*y, e = 1 - s2*y2, w0 = (gm*y)*y2,
//   w = w0 * (1 + e*(3/2 + 15/8 e))          [ (1-e)^(-3/2) to O(e^3) ~ 1e-19 ]
//   3 DFMA (accumulate, fixed ascending-j order per thread).
// The changeover test costs no FP64 instruction: for non-negative doubles
// hi32(s2) > hi32(rc2) implies s2 > rc2, so one integer compare of the high word of
// s2 against max(hi32(rcrit_i^2), max_{j in tile} hi32(rcrit_j^2)) proves K = 1; pairs
// that fail it (including the self pair, s2 = 0) take the exact slow path below.
#pragma once
#include "common.cuh"

namespace mopal {

struct AccelParams {
    const unsigned char* tiles;  // nTiles * ACC_TILE_BYTES, written by pack_kernel
    const double* x;             // 3*ld
    const double* rcrit;         // nb
    double* part;                // [nsplit][3][ld] partial sums
    int nb, ld, nTiles, tps;     // tps = tiles per j-split
};

// Exact K-weighted pair weight gm_j K / r^3 (readings A-1..A-5, A-9).  Rare path.
__device__ __noinline__ double slow_weight(double s2, double gmj, const double* __restrict__ rcrit, int i,
                                           int j, int nb) {
    if (i >= nb || j >= nb || !(s2 > 0.0)) return 0.0;
    double rc = fmax(rcrit[i], rcrit[j]);
    double s = sqrt(s2);
    double K = 1.0;
    if (s2 < rc * rc) {
        double rin = 0.1 * rc;
        if (s2 <= rin * rin) return 0.0;
        double q = (s - rin) / (0.9 * rc);
        K = q * q * q * (10.0 + q * (6.0 * q - 15.0));
    }
    return gmj * K / (s2 * s);
}

template <int IPT, int U>
__global__ void __launch_bounds__(CTA_THREADS) pair_accel_kernel(AccelParams p) {
    __shared__ __align__(128) unsigned char s_tiles[STAGES * ACC_TILE_BYTES];
    __shared__ __align__(8) uint64_t s_full[STAGES];
    __shared__ __align__(8) uint64_t s_empty[STAGES];

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int t0 = blockIdx.y * p.tps;
    const int nt = min(p.tps, p.nTiles - t0);

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; ++s) { mbar_init(&s_full[s], 1); mbar_init(&s_empty[s], CONSUMER_THREADS / 32); }
        mbar_fence_init();
    }
    __syncthreads();

    if (warp == CONSUMER_THREADS / 32) {  // ---- TMA producer warp ----
        if (lane == 0) {
            const unsigned char* src = p.tiles + (size_t)t0 * ACC_TILE_BYTES;
            for (int n = 0; n < nt; ++n) {
                const int st = n % STAGES;
                mbar_wait(&s_empty[st], ((n / STAGES) & 1) ^ 1);
                mbar_arrive_expect_tx(&s_full[st], ACC_TILE_BYTES);
                tma_load_1d(s_tiles + st * ACC_TILE_BYTES, src + (size_t)n * ACC_TILE_BYTES, ACC_TILE_BYTES,
                            &s_full[st]);
            }
        }
        return;
    }

    // ---- compute warps ----
    const int ibase = blockIdx.x * (CONSUMER_THREADS * IPT) + tid;
    double xi[IPT], yi[IPT], zi[IPT], ax[IPT], ay[IPT], az[IPT];
    int gi[IPT];
#pragma unroll
    for (int k = 0; k < IPT; ++k) {
        const int i = ibase + k * CONSUMER_THREADS;
        if (i < p.nb) {
            xi[k] = p.x[i]; yi[k] = p.x[p.ld + i]; zi[k] = p.x[2 * p.ld + i];
            const double rc = p.rcrit[i];
            gi[k] = __double2hiint(rc * rc);
        } else {
            xi[k] = yi[k] = zi[k] = 0.0; gi[k] = 0;
        }
        ax[k] = ay[k] = az[k] = 0.0;
    }

    for (int n = 0; n < nt; ++n) {
        const int st = n % STAGES;
        mbar_wait(&s_full[st], (n / STAGES) & 1);
        const unsigned char* tile = s_tiles + st * ACC_TILE_BYTES;
        const double2* tj = reinterpret_cast<const double2*>(tile);
        const int gt = *reinterpret_cast<const int*>(tile + TJ * 32);
        int g[IPT];
#pragma unroll
        for (int k = 0; k < IPT; ++k) g[k] = max(gi[k], gt);

#pragma unroll 1
        for (int jj = 0; jj < TJ; jj += U) {
            double dx[U][IPT], dy[U][IPT], dz[U][IPT], w[U][IPT];
            bool any = false;
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const double2 pa = tj[2 * (jj + u)];      // x, y
                const double2 pb = tj[2 * (jj + u) + 1];  // z, gm
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
                    any |= (__double2hiint(s2) <= g[k]);
                    dx[u][k] = ddx; dy[u][k] = ddy; dz[u][k] = ddz;
                }
            }
            if (any) {  // rare: changeover shell, self pair, coincident bodies
                const int jg = (t0 + n) * TJ + jj;
#pragma unroll
                for (int u = 0; u < U; ++u) {
#pragma unroll
                    for (int k = 0; k < IPT; ++k) {
                        const double s2 = fma(dz[u][k], dz[u][k], fma(dy[u][k], dy[u][k], dx[u][k] * dx[u][k]));
                        if (__double2hiint(s2) <= g[k])
                            w[u][k] = slow_weight(s2, tj[2 * (jj + u) + 1].y, p.rcrit,
                                                  ibase + k * CONSUMER_THREADS, jg + u, p.nb);
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
        __syncwarp();
        if (lane == 0) mbar_arrive(&s_empty[st]);
    }

    double* out = p.part + (size_t)blockIdx.y * 3 * p.ld;
#pragma unroll
    for (int k = 0; k < IPT; ++k) {
        const int i = ibase + k * CONSUMER_THREADS;
        if (i < p.nb) { out[i] = ax[k]; out[p.ld + i] = ay[k]; out[2 * p.ld + i] = az[k]; }
    }
}

// Partial sums -> a, in fixed split order; optionally the closing half kick
// v += hk * a (Hamiltonian block LOOP 1).
template <bool KICK>
__global__ void __launch_bounds__(ON_BLOCK) accel_reduce_kernel(const double* __restrict__ part, int nsplit,
                                                                 int nb, int ld, double* __restrict__ a,
                                                                 double* __restrict__ v, double hk) {
    const int i = blockIdx.x * ON_BLOCK + threadIdx.x;
    if (i >= nb) return;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        double s = 0.0;
        for (int sp = 0; sp < nsplit; ++sp) s += part[((size_t)sp * 3 + c) * ld + i];
        a[(size_t)c * ld + i] = s;
        if (KICK) v[(size_t)c * ld + i] = fma(hk, s, v[(size_t)c * ld + i]);
    }
}

// Builds the j-tiles {x,y,z,gm} + gate header from the SoA state; with JUMP it first
// applies the stellar jump x += hj * P / mu (Hamiltonian block LOOP 2-3,
// PAPER.md:209-219) using the block partial sums of gm*v.
constexpr double PAD_POS = 1.0e15;  // pad bodies: far away and massless -> contribute exactly 0

// Sum of gm v (Hamiltonian block LOOP 2): every block of the producing kernel
// writes a partial; the block that arrives last (ticket counter) adds the partials in index order
// - the same order whichever block that is - into psum[3 npsum ..], which the next kernel reads.
template <int BLOCK>
__device__ __forceinline__ void psum_finalize(double* psum, int npsum, unsigned* ticket, double (*sh)[3]) {
    __shared__ bool s_last;
    if (threadIdx.x == 0) {
        __threadfence();                                   // the partial is visible before the ticket
        s_last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    double s0 = 0, s1 = 0, s2 = 0;
    for (int b = threadIdx.x; b < npsum; b += BLOCK) {
        s0 += __ldcg(psum + 3 * b); s1 += __ldcg(psum + 3 * b + 1); s2 += __ldcg(psum + 3 * b + 2);
    }
    block_sum3<BLOCK>(s0, s1, s2, sh);
    if (threadIdx.x == 0) {
        psum[3 * npsum] = s0; psum[3 * npsum + 1] = s1; psum[3 * npsum + 2] = s2;
        *ticket = 0u;                                      // ready for the next launch
    }
}
__device__ __forceinline__ void load_psum(const double* __restrict__ psum, int npsum, double& P0, double& P1, double& P2) {
    P0 = psum[3 * npsum]; P1 = psum[3 * npsum + 1]; P2 = psum[3 * npsum + 2];
}

// SYM selects the tile layout: false = TJ records {x,y,z,gm} (pair_accel_kernel, broadcast reads),
// true = SoA halves {x,y}[TJ] then {z,gm}[TJ] (pair_sym_kernel, lane-distinct reads).
// nsrc = number of gravity sources (the big bodies): only the tiles that hold a
// source are written, and bodies j >= nsrc in the last of them become pad records.  The jump
// still moves every body (grid = all nb tiles with JUMP, the source tiles without).
template <bool JUMP, bool SYM>
__global__ void __launch_bounds__(TJ) pack_kernel(double* __restrict__ x, const double* __restrict__ gm,
                                                  const double* __restrict__ rcrit, int nb, int nsrc, int ld,
                                                  unsigned char* __restrict__ tiles,
                                                  const double* __restrict__ psum, int npsum, double hj_over_mu, Gate gate) {
    __shared__ int sg[TJ / 32];
    if (gate_closed(gate)) return;
    double sx = 0, sy = 0, sz = 0;
    if (JUMP) {
        double P0, P1, P2;
        load_psum(psum, npsum, P0, P1, P2);
        sx = hj_over_mu * P0; sy = hj_over_mu * P1; sz = hj_over_mu * P2;
    }
    const int j = blockIdx.x * TJ + threadIdx.x;
    double2 pa, pb;
    int ghi = 0;
    if (j < nb) {
        double X = x[j], Y = x[ld + j], Z = x[2 * ld + j];
        if (JUMP) {
            X += sx; Y += sy; Z += sz;
            x[j] = X; x[ld + j] = Y; x[2 * ld + j] = Z;
        }
        pa = make_double2(X, Y);
        pb = make_double2(Z, 0.0);
        if (j < nsrc) {
            pb.y = gm[j];
            const double rc = rcrit[j];
            ghi = __double2hiint(rc * rc);
        }
    }
    if (blockIdx.x * TJ >= nsrc) return;      // no source in this tile (block-uniform)
    if (j >= nsrc) {
        pa = make_double2(PAD_POS, PAD_POS);
        pb = make_double2(PAD_POS, 0.0);
    }
    unsigned char* tile = tiles + (size_t)blockIdx.x * (SYM ? SYM_TILE_BYTES : ACC_TILE_BYTES);
    if (SYM) {
        double2* rec = reinterpret_cast<double2*>(tile);
        rec[threadIdx.x] = pa; rec[TJ + threadIdx.x] = pb;
        reinterpret_cast<double*>(tile + SYM_RC_OFF)[threadIdx.x] = j < nsrc ? rcrit[j] : 0.0;
    } else {
        double2* rec = reinterpret_cast<double2*>(tile) + 2 * threadIdx.x;
        rec[0] = pa; rec[1] = pb;
    }
    ghi = __reduce_max_sync(0xffffffffu, ghi);
    if ((threadIdx.x & 31) == 0) sg[threadIdx.x >> 5] = ghi;
    __syncthreads();
    if (threadIdx.x == 0) {
        int g = sg[0];
#pragma unroll
        for (int k = 1; k < TJ / 32; ++k) g = max(g, sg[k]);
        int4 hdr = make_int4(g, 0, 0, 0);
        *reinterpret_cast<int4*>(tile + TJ * 32) = hdr;
    }
}

}  // namespace mopal
