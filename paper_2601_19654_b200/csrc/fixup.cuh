// fixup.cuh - lets the close-encounter solve (resolve.cuh) run BESIDE the O(N^2) pair sum instead of before it.
//
// In the resolving step (S-1 with readings X-1..X-6) the closing accelerations a(x) need the positions the
// encounter solve delivers - but the solve only moves the flagged bodies (the endpoints of the encounter pair list,
// ~1 % of the bodies: PAPER.md:122), and the stellar jump that follows is one common shift, which no pair separation
// sees.  So the pair sum is taken over the DRIFTED positions x1 while the solve runs (a chain of dependent right-hand
// sides on one SM, resolve.cuh), and afterwards, with F = the flagged bodies:
//     i not in F:  a_i += sum_{f in F} gm_f [ w(x_f - x_i) (x_f - x_i)  -  w(x1_f - x_i) (x1_f - x_i) ]     (fix_unflagged_kernel)
//     f in F:      a_f  = sum_{j != f} gm_j w(x_j - x_f) (x_j - x_f)   over all j, resolved positions      (fix_flagged_kernel)
// with w = K(r; max(rcrit_i, rcrit_j)) / r^3 (readings A-1..A-5, A-9) - 3 nb |F| pair evaluations, ~3 % of the pair sum at
// the headline config.  A removed term is recomputed, not remembered: it equals the term inside a_i to a few ulp of
// itself, far inside the 1e-12 sum|terms| tolerance.  Then the jump and the closing kick (jump_kick_kernel).
// Fixed orders everywhere (the flagged list is ascending): bit-reproducible.
#pragma once
#include "common.cuh"
#include "pair_accel.cuh"
#include "pair_sym.cuh"

namespace mopal {

constexpr int FIX_THREADS = 256;
constexpr int FIX_LIST_THREADS = 1024;

// exclusive block scan of one int per thread (up to 1024 threads)
__device__ __forceinline__ int fix_scan(int v, int* sScan, int& total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int incl = v;
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
    total = sScan[63];
    return (warp ? sScan[32 + warp - 1] : 0) + incl - v;
}

// F in ascending order: one CTA, thread t takes the bodies [t seg, (t+1) seg), seg a multiple of 8 (the flags are read
// eight at a time: almost all of them are 0)
__global__ void __launch_bounds__(FIX_LIST_THREADS) fix_list_kernel(const uint8_t* __restrict__ flag, int nb,
                                                                    int* __restrict__ flist, int* __restrict__ nf, Gate gate) {
    __shared__ int sScan[64];
    if (gate_closed(gate)) return;
    const int tid = threadIdx.x;
    const int seg = ((nb + FIX_LIST_THREADS - 1) / FIX_LIST_THREADS + 7) & ~7;
    const int b0 = min(nb, tid * seg), b1 = min(nb, b0 + seg);
    const bool wide = (reinterpret_cast<uintptr_t>(flag) & 7u) == 0;
    int cnt = 0;
    for (int b = b0; b < b1; b += 8) {
        if (wide && b + 8 <= b1 && *reinterpret_cast<const unsigned long long*>(flag + b) == 0ull) continue;
        const int e = min(b + 8, b1);
        for (int q = b; q < e; ++q) cnt += flag[q] ? 1 : 0;
    }
    int tot;
    int k = fix_scan(cnt, sScan, tot);
    if (cnt > 0)
        for (int b = b0; b < b1; ++b)
            if (flag[b]) flist[k++] = b;
    if (tid == 0) *nf = tot;
}

struct FixParams {
    const double* x;       // 3*ld: positions after the encounter solve (before the jump)
    const double* x1;      // 3*ld: drifted positions the pair sum was taken over
    const double* gm;      // nb
    const double* rcrit;   // nb
    const uint8_t* flag;   // nb
    const int* flist;      // F, ascending
    const int* nf;
    double* a;             // 3*ld in/out
    double* part;          // FIX_JS * 3 * nb: partial rows of the flagged bodies
    int nb, ld;
    Gate gate;
};

// K(r; rc) / r^3: outside the changeover radius (almost every pair) the seed + one third-order correction of the pair
// kernels, 9 FP64 instructions; else the exact path
__device__ __forceinline__ double fix_w(double s2, double rc) {
    if (s2 >= rc * rc && s2 > 0.0) {
        const double y = rsqrt_seed(s2);
        const double y2 = y * y;
        const double e = fma(-s2, y2, 1.0);
        const double u0 = y * y2;
        return fma(u0, e * fma(1.875, e, 1.5), u0);
    }
    return sym_slow_u(s2, rc);
}

constexpr int FIX_CHUNK = 256;   // flagged bodies staged per pass of fix_unflagged_kernel
constexpr int FIX_FB = 4;        // flagged bodies per CTA of fix_flagged_kernel
constexpr int FIX_JS = 8;        // j splits of a flagged body's row

constexpr int FIX_UT = 256;      // threads of fix_unflagged_kernel
constexpr int FIX_SP = 4;        // lanes that share a body there (measured at cfg3, 725 flagged bodies: 128 threads x 1 lane
                                 // 225 us, 128 x 2 201, 128 x 4 198, 256 x 4 187, 256 x 8 203)
__global__ void __launch_bounds__(FIX_UT) fix_unflagged_kernel(FixParams p) {
    __shared__ double sN[3][FIX_CHUNK], sO[3][FIX_CHUNK], sG[FIX_CHUNK], sR[FIX_CHUNK];
    if (gate_closed(p.gate)) return;
    const int nf = *p.nf;
    if (nf == 0) return;
    // FIX_SP neighbouring lanes share a body and take every FIX_SP-th flagged body of a chunk: more warps per SM for the
    // same staging (one warp in flight per 8 cycles of FP64 latency and sub-partition was not enough)
    const int i = blockIdx.x * (FIX_UT / FIX_SP) + threadIdx.x / FIX_SP, h = threadIdx.x % FIX_SP;
    const bool mine = i < p.nb && !p.flag[i];
    double xi = 0.0, yi = 0.0, zi = 0.0, rci = 0.0;
    if (mine) { xi = p.x[i]; yi = p.x[p.ld + i]; zi = p.x[2 * p.ld + i]; rci = p.rcrit[i]; }
    double c0 = 0.0, c1 = 0.0, c2 = 0.0;
    for (int base = 0; base < nf; base += FIX_CHUNK) {
        const int m = min(FIX_CHUNK, nf - base);
        __syncthreads();
        for (int t = threadIdx.x; t < m; t += FIX_UT) {
            const int f = p.flist[base + t];
#pragma unroll
            for (int c = 0; c < 3; ++c) { sN[c][t] = p.x[(size_t)c * p.ld + f]; sO[c][t] = p.x1[(size_t)c * p.ld + f]; }
            sG[t] = p.gm[f]; sR[t] = p.rcrit[f];
        }
        __syncthreads();
        if (mine) {
#pragma unroll 4
            for (int t = h; t < m; t += FIX_SP) {
                const double g = sG[t];
                const double rc = fmax(rci, sR[t]);
                const double nx = sN[0][t] - xi, ny = sN[1][t] - yi, nz = sN[2][t] - zi;
                const double ox = sO[0][t] - xi, oy = sO[1][t] - yi, oz = sO[2][t] - zi;
                const double un = g * fix_w(fma(nz, nz, fma(ny, ny, nx * nx)), rc);
                const double uo = g * fix_w(fma(oz, oz, fma(oy, oy, ox * ox)), rc);
                c0 += fma(un, nx, -(uo * ox)); c1 += fma(un, ny, -(uo * oy)); c2 += fma(un, nz, -(uo * oz));
            }
        }
    }
#pragma unroll
    for (int o = 1; o < FIX_SP; o <<= 1) {                 // the sharing lanes' sums, in a fixed order
        c0 += __shfl_xor_sync(0xffffffffu, c0, o); c1 += __shfl_xor_sync(0xffffffffu, c1, o); c2 += __shfl_xor_sync(0xffffffffu, c2, o);
    }
    if (mine && h == 0) { p.a[i] += c0; p.a[p.ld + i] += c1; p.a[2 * p.ld + i] += c2; }
}

// rows of the flagged bodies over the resolved positions: CTA (g, js) sums FIX_FB rows over the js-th part of the bodies j
// (every j loaded once for FIX_FB rows), fixed-order block sum -> part[js][f][c]
// (measured at cfg3, 725 flagged bodies: 8 rows per CTA at 169 registers - one CTA per SM - 154 us; 4 rows and two CTAs per
// SM 109 us; 2 rows 164 us)
__global__ void __launch_bounds__(FIX_THREADS, 2) fix_flagged_kernel(FixParams p) {
    __shared__ double sh[FIX_THREADS / 32][3 * FIX_FB];
    if (gate_closed(p.gate)) return;
    const int nf = *p.nf;
    const int js = blockIdx.y;
    for (int k0 = blockIdx.x * FIX_FB; k0 < nf; k0 += gridDim.x * FIX_FB) {
    int f[FIX_FB];
    double xf[FIX_FB], yf[FIX_FB], zf[FIX_FB], rcf[FIX_FB], s[FIX_FB][3];
#pragma unroll
    for (int r = 0; r < FIX_FB; ++r) {
        f[r] = k0 + r < nf ? p.flist[k0 + r] : -1;
        const int b = f[r] >= 0 ? f[r] : 0;
        xf[r] = p.x[b]; yf[r] = p.x[p.ld + b]; zf[r] = p.x[2 * p.ld + b]; rcf[r] = p.rcrit[b];
        s[r][0] = s[r][1] = s[r][2] = 0.0;
    }
    const int per = ((p.nb + FIX_JS - 1) / FIX_JS + FIX_THREADS - 1) / FIX_THREADS * FIX_THREADS;
    const int j0 = js * per, j1 = min(p.nb, j0 + per);
    // the next body's record is loaded while the current one is used
    int j = j0 + threadIdx.x;
    double nx = 0.0, ny = 0.0, nz = 0.0, ng = 0.0, nr = 0.0;
    if (j < j1) { nx = p.x[j]; ny = p.x[p.ld + j]; nz = p.x[2 * p.ld + j]; ng = p.gm[j]; nr = p.rcrit[j]; }
    for (; j < j1; j += FIX_THREADS) {
        const double xj = nx, yj = ny, zj = nz, gj = ng, rcj = nr;
        const int jn = j + FIX_THREADS;
        if (jn < j1) { nx = p.x[jn]; ny = p.x[p.ld + jn]; nz = p.x[2 * p.ld + jn]; ng = p.gm[jn]; nr = p.rcrit[jn]; }
#pragma unroll
        for (int r = 0; r < FIX_FB; ++r) {
            const double dx = xj - xf[r], dy = yj - yf[r], dz = zj - zf[r];
            const double u = gj * fix_w(fma(dz, dz, fma(dy, dy, dx * dx)), fmax(rcf[r], rcj));   // j = f: s2 = 0 -> 0
            s[r][0] = fma(u, dx, s[r][0]); s[r][1] = fma(u, dy, s[r][1]); s[r][2] = fma(u, dz, s[r][2]);
        }
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int r = 0; r < FIX_FB; ++r) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            double v = s[r][c];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
            if (lane == 0) sh[warp][3 * r + c] = v;
        }
    }
    __syncthreads();
    if (threadIdx.x < 3 * FIX_FB) {
        double t = 0.0;
#pragma unroll
        for (int w = 0; w < FIX_THREADS / 32; ++w) t += sh[w][threadIdx.x];
        const int r = threadIdx.x / 3, c = threadIdx.x - 3 * r;
        if (k0 + r < nf) p.part[((size_t)js * p.nb + (k0 + r)) * 3 + c] = t;
    }
    __syncthreads();                                      // sh free for the next group of rows
    }
}

__global__ void __launch_bounds__(FIX_THREADS) fix_flagged_reduce_kernel(FixParams p) {
    if (gate_closed(p.gate)) return;
    const int nf = *p.nf;
    const int k = blockIdx.x * FIX_THREADS + threadIdx.x;
    if (k >= nf) return;
    const int f = p.flist[k];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        double t = 0.0;
#pragma unroll
        for (int js = 0; js < FIX_JS; ++js) t += p.part[((size_t)js * p.nb + k) * 3 + c];
        p.a[(size_t)c * p.ld + f] = t;
    }
}

// second jump x += hj P / mu (Hamiltonian block LOOP 2-3) and closing kick v += hk a (LOOP 1)
__global__ void __launch_bounds__(ON_BLOCK) jump_kick_kernel(double* __restrict__ x, double* __restrict__ v,
                                                              const double* __restrict__ a, const double* __restrict__ psum,
                                                              int npsum, double hj_over_mu, double hk, int nb, int ld, Gate gate) {
    if (gate_closed(gate)) return;
    const int b = blockIdx.x * ON_BLOCK + threadIdx.x;
    if (b >= nb) return;
    double P0, P1, P2;
    load_psum(psum, npsum, P0, P1, P2);
    x[b] += hj_over_mu * P0; x[ld + b] += hj_over_mu * P1; x[2 * ld + b] += hj_over_mu * P2;
    v[b] = fma(hk, a[b], v[b]); v[ld + b] = fma(hk, a[ld + b], v[ld + b]); v[2 * ld + b] = fma(hk, a[2 * ld + b], v[2 * ld + b]);
}

// the step's way of getting its accelerations: taken over from what the last step's label kernel saw
__global__ void mode_latch_kernel(int* mode) { mode[0] = mode[1]; }

}  // namespace mopal
