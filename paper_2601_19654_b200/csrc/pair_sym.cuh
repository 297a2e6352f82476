// pair_sym.cuh - two-sided ("Newton III") form of the O(N^2) K(r)-weighted mutual-gravity
// sum (force block LOOP 2):  a_i = sum_{j != i} gm_j K_ij (x_j - x_i) / r_ij^3.
//
// K_ij = K_ji (rc = max(rcrit_i, rcrit_j), reading A-3), so u_ij = K_ij / r_ij^3 is evaluated once
// per UNORDERED pair and applied to both bodies:  a_i += gm_j u d,  a_j -= gm_i u d,  d = x_j - x_i.
// FP64-pipe cost per unordered pair on the K = 1 path: 3 DADD (d), DMUL + 2 DFMA (s2), 4 DMUL +
// 3 DFMA (u from the MUFU.RSQ64H seed, one third-order correction), 2 DMUL (gm_j u, gm_i u),
// 6 DFMA (two accumulations) = 20, i.e. 10 per ordered pair against 16 for the one-sided kernel.
//
// Work unit = (row block I of SYM_R = 128*IPT bodies) x (a chunk of j tiles at or right of the
// block's diagonal; the units at the end of the list are cut finer - single tiles, then single groups of 32 bodies of
// a tile - so that the CTAs of the last wave end together, see plan_sym_units in mopal.cu).  Each lane keeps IPT bodies
// i resident (position, gm, gate, accumulators).
// A j tile is 4 groups of 32 bodies; a group ROTATES through the warp: at rotation s lane L works
// on j = (L + s) mod 32, reading its record from the shared-memory tile (SoA halves {x,y}[128] and
// {z,gm}[128]: 16-byte stride, conflict-free for lane-distinct addresses) and carrying the three
// accumulators of that j in registers, handed to the neighbouring lane by SHFL after every
// rotation (6 SHFL.32 per 120 FP64 instructions at IPT = 6).  After 32 rotations every lane holds the partial
// a_j of its home j = L.  The 4 warps' partials are combined through shared memory in warp order
// and written to a triangular partial buffer partJ[I][c][j >= I*SYM_R]; the resident a_i go to
// partI[unit][c][row].  sym_reduce_kernel adds, for each body, its row partials in unit order and
// then its column partials in ascending I: a fixed tree that depends on nb only (reading A-8) -
// no atomics, bit-reproducible.
//
// Diagonal tiles (j tile inside the row block) take each unordered pair once by masking j <= i (at IPT = 6 a warp skips the
// groups of 32 columns that lie wholly below its rows: three quarters of the masked work).
// Changeover / coincident pairs are caught by the same integer gate as in pair_accel.cuh (here one
// compare per rotation: min of the IPT high words of s2 against the largest gate of the lane's
// bodies and of the tile) and recomputed exactly by slow_weight(gm = 1).
//
// Tuning record (B200, N = 65,536; the SYM_* macros exist for these sweeps): IPT 4 at 3 CTAs/SM
// 2.92 ms, IPT 6 at 2 CTAs/SM 2.87 ms, IPT 7 2.97 ms, IPT 8 spills; more resident warps do not help
// (the FP64 pipe, not latency, is the limit: a pure DFMA stream reaches 86-90 % of the nominal peak
// on this chip, every non-FP64 instruction costs about one more issue cycle); an FP32 MUFU.RSQ seed
// re-biased with integer instructions is slower than MUFU.RSQ64H (+8 %).
#pragma once
#include "common.cuh"
#include "pair_accel.cuh"

namespace mopal {

#ifndef SYM_STAGES_N
#define SYM_STAGES_N 4
#endif
constexpr int SYM_STAGES = SYM_STAGES_N;
// Bodies i per lane (IPT): a template parameter - 6 for the large systems (768-row blocks: least shuffle traffic per
// FP64 instruction), 3 and 2 for the mid-size ones, whose triangle would otherwise break into too few, too long work
// units for the 148 SMs (a unit of IPT x 128 rows by one 128-body tile is 256 IPT pair evaluations per lane).
// A row block spans IPT j tiles (128 IPT rows).
__host__ __device__ constexpr int sym_rows(int ipt) { return CONSUMER_THREADS * ipt; }

struct SymParams {
    const unsigned char* tiles;  // nTiles * SYM_TILE_BYTES, SoA-planes layout (pack_kernel<.., true>)
    const double* x;             // 3*ld
    const double* gm;            // nb
    const double* rcrit;         // nb
    const int4* units;           // {I, t0, t1, g0 | g1 << 8}: j tiles [t0, t1) of row block I; of a single tile, the
                                 // groups of 32 bodies [g0, g1) (all four of every tile of a longer unit)
    double* partI;               // [nUnits][3][R], R = 128 IPT
    double* partJ;               // triangular: block I at symJ_off(I), planes of (nbPad - I*R)
    int nb, ld, nbPad;
    int unit0;                   // first work unit of this launch (a rank's share of the units, row f4; 0 otherwise)
    Gate gate;
};

__host__ __device__ inline long long symJ_off(int I, int nbPad, int R) {
    return 3LL * ((long long)I * nbPad - (long long)R * ((long long)I * (I - 1) / 2));
}

// Tile of the two-sided kernel: {x,y}[128] | {z,gm}[128] | 16 B header (largest changeover gate of the tile) | rcrit[128]
// (the last plane is read on the changeover path only: no global load there)
constexpr int SYM_TILE_STRIDE = 5632;   // shared-memory stage stride: tile padded to 11 x 512 B

__device__ __forceinline__ void lds_rec(double2& a, double2& b, uint32_t addr) {
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(a.x), "=d"(a.y) : "r"(addr));
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2+2048];" : "=d"(b.x), "=d"(b.y) : "r"(addr));
}

// next record of the 32-record (512 B, 512-B aligned) group, cyclically: VIADD + one LOP3
__device__ __forceinline__ uint32_t next_rec(uint32_t addr) { return (addr & ~511u) | ((addr + 16u) & 511u); }

// K(r; rc) / r^3 of a pair that may be inside a changeover shell (readings A-1..A-5, A-9), from registers and shared
// memory alone: a giant's row or tile sends thousands of pairs here, so there is no function call, no global load and
// no square root (the refined MUFU seed, 2 ulp) - one division, for the pairs that really are inside the shell.
__device__ __forceinline__ double sym_slow_u(double s2, double rc) {
    if (!(s2 > 0.0)) return 0.0;                       // coincident bodies, self pairs
    const double y0 = rsqrt_seed(s2);
    const double e = fma(-s2, y0 * y0, 1.0);
    const double y = fma(y0, e * fma(0.375, e, 0.5), y0);
    const double y3 = y * (y * y);
    if (s2 >= rc * rc) return y3;                      // K = 1
    const double rin = 0.1 * rc;
    if (s2 <= rin * rin) return 0.0;                   // K = 0
    const double q = (s2 * y - rin) / (0.9 * rc);
    return q * q * q * (10.0 + q * (6.0 * q - 15.0)) * y3;
}

// one rotation: IPT pairs of this lane against the body whose record is (ca, cb).  The record of
// the NEXT rotation is loaded into (na, nb2) as soon as this rotation's separations are formed, so
// the shared-memory latency is covered by the FP64 instructions that follow.  An FP64 warp
// instruction holds the sub-partition's issue port for two cycles, so every other instruction
// costs half a DFMA: the changeover gate is ONE compare per rotation (min over the IPT high words
// of s2 against the largest gate of the lane's bodies and the tile), the j index is only formed on
// the slow path, and the records ping-pong between two register sets (no copies).
template <int SYM_IPT, bool DIAG>
__device__ __forceinline__ void sym_rotation(const double2 ca, const double2 cb, double2& na, double2& nb2,
                                             const uint32_t caddr, const uint32_t naddr, const int jgrp,
                                             const int ibase, const double (&xi)[SYM_IPT],
                                             const double (&yi)[SYM_IPT], const double (&zi)[SYM_IPT],
                                             const double (&mi)[SYM_IPT], const int g,
                                             double (&ax)[SYM_IPT], double (&ay)[SYM_IPT], double (&az)[SYM_IPT],
                                             double& tx, double& ty, double& tz, const double (&rci)[SYM_IPT],
                                             const uint32_t rcbase, const double* __restrict__ rcrit, int nb) {
    double dx[SYM_IPT], dy[SYM_IPT], dz[SYM_IPT], u[SYM_IPT];
#pragma unroll
    for (int k = 0; k < SYM_IPT; ++k) {
        dx[k] = ca.x - xi[k]; dy[k] = ca.y - yi[k]; dz[k] = cb.x - zi[k];
    }
    lds_rec(na, nb2, naddr);
    int hmin = 0x7fffffff;
#pragma unroll
    for (int k = 0; k < SYM_IPT; ++k) {
        const double s2 = fma(dz[k], dz[k], fma(dy[k], dy[k], dx[k] * dx[k]));
        const double y = rsqrt_seed(s2);
        const double y2 = y * y;
        const double e = fma(-s2, y2, 1.0);
        const double u0 = y * y2;
        const double t = e * fma(1.875, e, 1.5);
        u[k] = fma(u0, t, u0);
        hmin = min(hmin, __double2hiint(s2));
    }
    const int jglob_d = DIAG ? jgrp + (int)((caddr & 511u) >> 4) : 0;
    if (DIAG) {   // each unordered pair of a diagonal tile once: j > i only
#pragma unroll
        for (int k = 0; k < SYM_IPT; ++k) u[k] = jglob_d > ibase + k * 32 ? u[k] : 0.0;
    }
    if (hmin <= g) {  // a pair that may be inside a changeover shell, or coincident bodies
        const int jglob = jgrp + (int)((caddr & 511u) >> 4);
        if constexpr (SYM_IPT >= 6) {
            // large systems: a few of thousands of units meet a giant - the out-of-line path (two global loads) costs
            // nothing there, and the kernel keeps its registers for the six resident bodies
#pragma unroll
            for (int k = 0; k < SYM_IPT; ++k) {
                const double q2 = fma(dz[k], dz[k], fma(dy[k], dy[k], dx[k] * dx[k]));
                if (__double2hiint(q2) <= g && (!DIAG || jglob > ibase + k * 32))
                    u[k] = slow_weight(q2, 1.0, rcrit, ibase + k * 32, jglob, nb);
            }
        } else {
            // mid-size systems: the kernel is as long as its slowest unit, and the unit with a giant's row takes this
            // path in every rotation
            double rcj;
            asm volatile("ld.shared.f64 %0, [%1];" : "=d"(rcj) : "r"(rcbase + ((caddr & 511u) >> 1)));
#pragma unroll
            for (int k = 0; k < SYM_IPT; ++k) {
                const double q2 = fma(dz[k], dz[k], fma(dy[k], dy[k], dx[k] * dx[k]));
                if (__double2hiint(q2) <= g && (!DIAG || jglob > ibase + k * 32)) u[k] = sym_slow_u(q2, fmax(rci[k], rcj));
            }
        }
    }
#pragma unroll
    for (int k = 0; k < SYM_IPT; ++k) {
        const double wj = cb.y * u[k];
        const double wi = mi[k] * u[k];
        ax[k] = fma(wj, dx[k], ax[k]);
        ay[k] = fma(wj, dy[k], ay[k]);
        az[k] = fma(wj, dz[k], az[k]);
        tx = fma(-wi, dx[k], tx);
        ty = fma(-wi, dy[k], ty);
        tz = fma(-wi, dz[k], tz);
    }
}

// tile_sa: shared-space address of the tile (512-B aligned); records {x,y}[TJ] then {z,gm}[TJ]
template <int SYM_IPT, bool DIAG>
__device__ __forceinline__ void sym_tile(const uint32_t tile_sa, const int jbase, const int lane, const int ibase,
                                         const double (&xi)[SYM_IPT], const double (&yi)[SYM_IPT],
                                         const double (&zi)[SYM_IPT], const double (&mi)[SYM_IPT],
                                         const int g, double (&ax)[SYM_IPT], double (&ay)[SYM_IPT],
                                         double (&az)[SYM_IPT], double* __restrict__ sj,
                                         const double (&rci)[SYM_IPT], const double* __restrict__ rcrit, int nb,
                                         const int g0, const int g1) {
    const unsigned full = 0xffffffffu;
#pragma unroll 1
    for (int grp = g0; grp < g1; ++grp) {
        // this lane walks the group's 32 records cyclically, starting at its home record
        uint32_t a0 = tile_sa + grp * 512 + lane * 16;
        const int jgrp = jbase + grp * 32;
        if (DIAG && SYM_IPT >= 6 && jgrp + 31 <= ibase - lane) {   // every j of the group <= every i of this warp: nothing to take
            // (the large systems only: -0.8 % at N = 65,536; the mid-size kernels measured 1.5 % slower with the test)
            sj[grp * 32 + lane] = 0.0; sj[TJ + grp * 32 + lane] = 0.0; sj[2 * TJ + grp * 32 + lane] = 0.0;
            continue;
        }
        const uint32_t rcbase = tile_sa + SYM_RC_OFF + grp * 256;
        double tx = 0.0, ty = 0.0, tz = 0.0;
        double2 pa, pb, qa, qb;
        lds_rec(pa, pb, a0);
#pragma unroll 1
        for (int s = 0; s < 32; s += 2) {
            const uint32_t a1 = next_rec(a0);
            sym_rotation<SYM_IPT, DIAG>(pa, pb, qa, qb, a0, a1, jgrp, ibase, xi, yi, zi, mi, g, ax, ay, az, tx, ty, tz, rci,
                               rcbase, rcrit, nb);
            // hand the travelling sums of j = (lane+s) to the lane that works on that j next
            tx = __shfl_sync(full, tx, lane + 1);
            ty = __shfl_sync(full, ty, lane + 1);
            tz = __shfl_sync(full, tz, lane + 1);
            a0 = next_rec(a1);                             // s = 30 wraps to the home record (unused load)
            sym_rotation<SYM_IPT, DIAG>(qa, qb, pa, pb, a1, a0, jgrp, ibase, xi, yi, zi, mi, g, ax, ay, az, tx, ty, tz, rci,
                               rcbase, rcrit, nb);
            tx = __shfl_sync(full, tx, lane + 1);
            ty = __shfl_sync(full, ty, lane + 1);
            tz = __shfl_sync(full, tz, lane + 1);
        }
        // after 32 rotations lane L holds the sums of its home j = grp*32 + L
        sj[grp * 32 + lane] = tx;
        sj[TJ + grp * 32 + lane] = ty;
        sj[2 * TJ + grp * 32 + lane] = tz;
    }
}

// No producer warp here: after the per-tile barrier every warp is done with the tile's slot, so
// thread 0 refills it (TMA 1-D bulk copy, completion on the slot's mbarrier) - 128 threads x 168
// registers lets 3 CTAs = 12 compute warps share an SM.
constexpr int SYM_THREADS = CONSUMER_THREADS;

template <int SYM_IPT>
__global__ void __launch_bounds__(SYM_THREADS, SYM_IPT >= 5 ? 2 : SYM_IPT >= 3 ? 3 : 4) pair_sym_kernel(SymParams p) {
    constexpr int SYM_R = sym_rows(SYM_IPT), SYM_TPB = SYM_IPT;
    constexpr int LOAD_BYTES = SYM_IPT >= 6 ? ACC_TILE_BYTES : SYM_TILE_BYTES;   // the rcrit plane is read by the in-line changeover path only
    __shared__ __align__(512) unsigned char s_tiles[SYM_STAGES * SYM_TILE_STRIDE];
    __shared__ __align__(16) double s_aj[2][SYM_THREADS / 32][3 * TJ];   // [parity][warp][c][j]
    __shared__ __align__(8) uint64_t s_full[SYM_STAGES];

    if (gate_closed(p.gate)) return;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int ug = blockIdx.x + p.unit0;
    const int4 un = p.units[ug];
    const int I = un.x, t0 = un.y, nt = un.z - un.y;
    const int g0 = un.w & 0xff, g1 = un.w >> 8;
    const unsigned char* src = p.tiles + (size_t)t0 * SYM_TILE_BYTES;

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < SYM_STAGES; ++s) mbar_init(&s_full[s], 1);
        mbar_fence_init();
#pragma unroll
        for (int s = 0; s < SYM_STAGES; ++s) {
            if (s < nt) {
                mbar_arrive_expect_tx(&s_full[s], LOAD_BYTES);
                tma_load_1d(s_tiles + s * SYM_TILE_STRIDE, src + (size_t)s * SYM_TILE_BYTES, LOAD_BYTES, &s_full[s]);
            }
        }
    }
    __syncthreads();

    // ---- compute warps: resident bodies i = I*SYM_R + warp*32*IPT + k*32 + lane ----
    const int ibase = I * SYM_R + warp * (32 * SYM_IPT) + lane;
    double xi[SYM_IPT], yi[SYM_IPT], zi[SYM_IPT], mi[SYM_IPT], rci[SYM_IPT], ax[SYM_IPT], ay[SYM_IPT], az[SYM_IPT];
    int gi = 0;   // largest changeover gate of this lane's bodies: high word of rcrit_i^2
#pragma unroll
    for (int k = 0; k < SYM_IPT; ++k) {
        const int i = ibase + k * 32;
        if (i < p.nb) {
            xi[k] = p.x[i]; yi[k] = p.x[p.ld + i]; zi[k] = p.x[2 * p.ld + i];
            mi[k] = p.gm[i];
            const double rc = p.rcrit[i];
            rci[k] = rc;
            gi = max(gi, __double2hiint(rc * rc));
        } else {   // pad rows: far away and massless
            xi[k] = yi[k] = zi[k] = -PAD_POS; mi[k] = 0.0; rci[k] = 0.0;
        }
        ax[k] = ay[k] = az[k] = 0.0;
    }

    const int jrow0 = I * SYM_R;                       // first column of partJ block I
    const int jw = p.nbPad - jrow0;                    // its plane width
    double* pj = p.partJ + symJ_off(I, p.nbPad, SYM_R);

    for (int n = 0; n < nt; ++n) {
        const int st = n % SYM_STAGES;
        const int t = t0 + n;
        mbar_wait(&s_full[st], (n / SYM_STAGES) & 1);
        const unsigned char* tile = s_tiles + st * SYM_TILE_STRIDE;
        const uint32_t tile_sa = smem_u32(tile);
        const int gt = *reinterpret_cast<const int*>(tile + TJ * 32);
        const int g = max(gi, gt);
        double* sj = s_aj[n & 1][warp];
        if (t < (I + 1) * SYM_TPB)
            sym_tile<SYM_IPT, true>(tile_sa, t * TJ, lane, ibase, xi, yi, zi, mi, g, ax, ay, az, sj, rci, p.rcrit, p.nb, g0, g1);
        else
            sym_tile<SYM_IPT, false>(tile_sa, t * TJ, lane, ibase, xi, yi, zi, mi, g, ax, ay, az, sj, rci, p.rcrit, p.nb, g0, g1);
        // combine the 4 warps' column partials in warp order (double-buffered: one barrier per tile)
        __syncthreads();
        if (tid == 0 && n + SYM_STAGES < nt) {   // every warp has left slot st: refill it
            mbar_arrive_expect_tx(&s_full[st], LOAD_BYTES);
            tma_load_1d(s_tiles + st * SYM_TILE_STRIDE, src + (size_t)(n + SYM_STAGES) * SYM_TILE_BYTES, LOAD_BYTES,
                        &s_full[st]);
        }
        const int jc = t * TJ + tid - jrow0;
        if (warp >= g0 && warp < g1) {           // the columns this unit worked on (the others belong to its sister units)
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                double s = s_aj[n & 1][0][c * TJ + tid];
#pragma unroll
                for (int w = 1; w < SYM_THREADS / 32; ++w) s += s_aj[n & 1][w][c * TJ + tid];
                pj[(size_t)c * jw + jc] = s;
            }
        }
    }

    double* pi = p.partI + (size_t)ug * 3 * SYM_R;
#pragma unroll
    for (int k = 0; k < SYM_IPT; ++k) {
        const int r = warp * (32 * SYM_IPT) + k * 32 + lane;
        pi[r] = ax[k]; pi[SYM_R + r] = ay[k]; pi[2 * SYM_R + r] = az[k];
    }
}

// a_b = (row partials of b's block, in unit order) + (column partials, ascending I); optionally
// the closing half kick v += hk * a (Hamiltonian block LOOP 1).
// SHARD (the pair sum sharded over GPUs): only the work units [us0, us1) were run - a contiguous run of
// every row block's units, i.e. of its groups of 32 columns: qr[I] = {first, end} group of block I's columns, counted
// from the block's diagonal, that this rank worked on.  The sum over the ranks of the results is the full acceleration.
#ifndef RED_SLICES_N
#define RED_SLICES_N 8
#endif
constexpr int RED_SLICES = RED_SLICES_N;           // threads per (body, component) of sym_reduce_kernel
constexpr int RED_THREADS = 32 * RED_SLICES;       // a block: 32 consecutive bodies (one row block: SYM_R is a multiple of 32)
template <bool KICK, bool SHARD>
__global__ void __launch_bounds__(RED_THREADS) sym_reduce_kernel(const double* __restrict__ partI,
                                                                  const double* __restrict__ partJ,
                                                                  const int* __restrict__ ustart, int nb, int ld,
                                                                  int nbPad, double* __restrict__ a,
                                                                  double* __restrict__ v, double hk, int us0, int us1,
                                                                  const int2* __restrict__ qr, int SYM_R, Gate gate) {
    __shared__ double sh[RED_SLICES][32];
    if (gate_closed(gate)) return;
    // blockIdx.y = component; warp w of the block = slice w: it takes the units u0 + w, u0 + w + 8, ... of the body's row
    // block and the column partials of the row blocks I = w, w + 8, ... (two interleaved sums each), and warp 0 adds the
    // eight slices in slice order: a fixed tree that depends on nb only, with eight times the loads in flight of a
    // thread-per-body loop (a row block cut into single column groups has hundreds of units)
    const int lane = threadIdx.x & 31, sl = threadIdx.x >> 5;
    const int b = blockIdx.x * 32 + lane;
    const int c = blockIdx.y;
    const int SYM_TPB = SYM_R / TJ;
    double s = 0.0;
    if (b < nb) {
        const int Ib = b / SYM_R, r = b - Ib * SYM_R;
        const int u0 = SHARD ? max(ustart[Ib], us0) : ustart[Ib], u1 = SHARD ? min(ustart[Ib + 1], us1) : ustart[Ib + 1];
        double s0 = 0.0, s1 = 0.0;
        int u = u0 + sl;
        for (; u + RED_SLICES < u1; u += 2 * RED_SLICES) {
            s0 += partI[((size_t)u * 3 + c) * SYM_R + r];
            s1 += partI[((size_t)(u + RED_SLICES) * 3 + c) * SYM_R + r];
        }
        if (u < u1) s0 += partI[((size_t)u * 3 + c) * SYM_R + r];
        // the column partial of row block I was written by the unit(s) that hold this body's group of 32 columns
        const int qb = b >> 5;
        auto colpart = [&](int I) -> double {
            if (SHARD) {
                const int2 r2 = qr[I];
                const int q = qb - I * SYM_TPB * (TJ / 32);
                if (q < r2.x || q >= r2.y) return 0.0;
            }
            return partJ[symJ_off(I, nbPad, SYM_R) + (size_t)c * (nbPad - I * SYM_R) + (b - I * SYM_R)];
        };
        double t0 = 0.0, t1 = 0.0;
        int I = sl;
        for (; I + RED_SLICES <= Ib; I += 2 * RED_SLICES) { t0 += colpart(I); t1 += colpart(I + RED_SLICES); }
        if (I <= Ib) t0 += colpart(I);
        s = (s0 + s1) + (t0 + t1);
    }
    sh[sl][lane] = s;
    __syncthreads();
    if (sl == 0 && b < nb) {
        double tot = sh[0][lane];
#pragma unroll
        for (int w = 1; w < RED_SLICES; ++w) tot += sh[w][lane];
        a[(size_t)c * ld + b] = tot;
        if (KICK) v[(size_t)c * ld + b] = fma(hk, tot, v[(size_t)c * ld + b]);
    }
}

}  // namespace mopal
