// support.cuh - the per-step support routines the paper lists next to the hot path
// (PAPER.md:84-94), kept on the device so that a long run never leaves it (the paper computes the
// critical radii on the host and copies them in every step, PAPER.md:291 item 3):
//   vshift_kernel   mco_h2dh / mce_dh2h (PAPER.md:84 item 1, fn. 12): heliocentric <-> democratic
//                   heliocentric, i.e. v_j -= sum gm v / (mu + sum gm)  or  v_j += sum gm v / mu
//   hill_kernel     mce_hill + the critical radius of mce_init (fn. 14):
//                   r_H = d (gm / 3 mu)^(1/3), rcrit = n_hill r_H, d = |x| (instantaneous star-planet
//                   separation) or the osculating semi-major axis (variant)
//   energy_*        mxx_en: kinetic + potential energy and angular momentum of
//                   star + bodies in the barycentric frame
// Readings H-1..H-4, E-1..E-3 in DESIGN.md section 3.  Everything is in gm = G m units on the
// device (G E = 1/2 sum gm v^2 + ...); the host divides by G once.
#pragma once
#include "common.cuh"
#include "pair_accel.cuh"

namespace mopal {

// sum of gm, fixed order: one block, thread-strided partials, shuffle tree, warps in order
__global__ void __launch_bounds__(1024) gmsum_kernel(const double* __restrict__ gm, int nb, double* __restrict__ out) {
    __shared__ double sh[32];
    double s = 0.0;
    for (int b = threadIdx.x; b < nb; b += 1024) s += gm[b];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int k = 0; k < 32; ++k) t += sh[k];
        *out = t;
    }
}

// v_j += scale * P, P = sum gm v (finished by the producing kernel's last block);
// TO_DH: scale = -1 / (mu + sum gm)   (H-1), else scale = +1 / mu   (H-2)
template <bool TO_DH>
__global__ void __launch_bounds__(ON_BLOCK) vshift_kernel(double* __restrict__ v, const double* __restrict__ psum, int npsum,
                                                          const double* __restrict__ gmsum, double mu, int nb, int ld) {
    const int b = blockIdx.x * ON_BLOCK + threadIdx.x;
    if (b >= nb) return;
    double P0, P1, P2;
    load_psum(psum, npsum, P0, P1, P2);
    const double den = TO_DH ? mu + *gmsum : mu;
    const double sgn = TO_DH ? -1.0 : 1.0;
    v[b] += sgn * (P0 / den);
    v[ld + b] += sgn * (P1 / den);
    v[2 * ld + b] += sgn * (P2 / den);
}

// Hill radius of one body.  mode 0: d = |x| ; mode 1: d = osculating a from the heliocentric velocity
// v + P / mu, P = sum gm v (unbound: |x|)
__device__ __forceinline__ double hill_body(double X, double Y, double Z, double vx, double vy, double vz, double g,
                                            double mu, double P0, double P1, double P2, int mode) {
    double d = sqrt(fma(Z, Z, fma(Y, Y, X * X)));
    if (mode == 1) {
        const double hx = vx + P0 / mu, hy = vy + P1 / mu, hz = vz + P2 / mu;
        const double v2 = fma(hz, hz, fma(hy, hy, hx * hx));
        const double inva = 2.0 / d - v2 / (mu + g);
        if (inva > 0.0) d = 1.0 / inva;
    }
    return d * cbrt(g / (3.0 * mu));
}

template <int MODE>
__global__ void __launch_bounds__(ON_BLOCK) hill_kernel(const double* __restrict__ x, const double* __restrict__ v,
                                                        const double* __restrict__ gm, const double* __restrict__ psum,
                                                        int npsum, double mu, double nhill, int nb, int ld,
                                                        double* __restrict__ rcrit, double* __restrict__ rhill) {
    const int b = blockIdx.x * ON_BLOCK + threadIdx.x;
    if (b >= nb) return;
    double P0 = 0.0, P1 = 0.0, P2 = 0.0, vx = 0.0, vy = 0.0, vz = 0.0;
    if (MODE == 1) {
        load_psum(psum, npsum, P0, P1, P2);
        vx = v[b]; vy = v[ld + b]; vz = v[2 * ld + b];
    }
    const double rh = hill_body(x[b], x[ld + b], x[2 * ld + b], vx, vy, vz, gm[b], mu, P0, P1, P2, MODE);
    if (rhill) rhill[b] = rh;
    rcrit[b] = nhill * rh;
}

// ---- energy and angular momentum ---------------------------------------------------------------
constexpr int EN_NSUM = 8;     // per-block partials: sum gm v (3), 1/2 sum gm v^2, sum gm / r, sum gm x cross v (3)

__global__ void __launch_bounds__(ON_BLOCK) energy_on_kernel(const double* __restrict__ x, const double* __restrict__ v,
                                                             const double* __restrict__ gm, int nb, int ld,
                                                             double* __restrict__ part) {
    __shared__ double sh[ON_BLOCK / 32][EN_NSUM];
    const int b = blockIdx.x * ON_BLOCK + threadIdx.x;
    double s[EN_NSUM];
#pragma unroll
    for (int k = 0; k < EN_NSUM; ++k) s[k] = 0.0;
    if (b < nb) {
        const double X = x[b], Y = x[ld + b], Z = x[2 * ld + b];
        const double vx = v[b], vy = v[ld + b], vz = v[2 * ld + b];
        const double g = gm[b];
        s[0] = g * vx; s[1] = g * vy; s[2] = g * vz;
        s[3] = 0.5 * g * fma(vz, vz, fma(vy, vy, vx * vx));
        s[4] = g / sqrt(fma(Z, Z, fma(Y, Y, X * X)));
        s[5] = g * (Y * vz - Z * vy); s[6] = g * (Z * vx - X * vz); s[7] = g * (X * vy - Y * vx);
    }
#pragma unroll
    for (int k = 0; k < EN_NSUM; ++k) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s[k] += __shfl_down_sync(0xffffffffu, s[k], o);
    }
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) {
#pragma unroll
        for (int k = 0; k < EN_NSUM; ++k) sh[w][k] = s[k];
    }
    __syncthreads();
    if (threadIdx.x < EN_NSUM) {
        double t = 0.0;
#pragma unroll
        for (int k = 0; k < ON_BLOCK / 32; ++k) t += sh[k][threadIdx.x];
        part[(size_t)blockIdx.x * EN_NSUM + threadIdx.x] = t;
    }
}

// sum over the interacting pairs i < j, i < nbig, of gm_i gm_j / r_ij.  CTA (bi, s) owns EN_T bodies i
// and the j tiles bi + s, bi + s + gridDim.y, ...; 12 FP64-pipe instructions per pair on the MUFU seed
// + one third-order correction (as in the pair sum); coincident bodies contribute 0 (as in the oracle).
constexpr int EN_T = 256;
__global__ void __launch_bounds__(EN_T) energy_pair_kernel(const double* __restrict__ x, const double* __restrict__ gm,
                                                            int nb, int nbig, int ld, double* __restrict__ part) {
    __shared__ __align__(16) double2 s_j[2 * EN_T];
    __shared__ double sh[EN_T / 32];
    const int tid = threadIdx.x;
    const int i = blockIdx.x * EN_T + tid;
    const bool iok = i < nbig;
    const double xi = iok ? x[i] : 0.0, yi = iok ? x[ld + i] : 0.0, zi = iok ? x[2 * ld + i] : 0.0;
    double acc = 0.0;
    const int nT = (nb + EN_T - 1) / EN_T;
    for (int t = blockIdx.x + blockIdx.y; t < nT; t += gridDim.y) {
        __syncthreads();
        const int j = t * EN_T + tid;
        if (j < nb) {
            s_j[2 * tid] = make_double2(x[j], x[ld + j]);
            s_j[2 * tid + 1] = make_double2(x[2 * ld + j], gm[j]);
        } else {
            s_j[2 * tid] = make_double2(PAD_POS, PAD_POS);
            s_j[2 * tid + 1] = make_double2(PAD_POS, 0.0);
        }
        __syncthreads();
        const int jlo = (t == blockIdx.x) ? tid + 1 : 0;      // diagonal tile: j > i only
#pragma unroll 4
        for (int jj = 0; jj < EN_T; ++jj) {
            const double2 pa = s_j[2 * jj], pb = s_j[2 * jj + 1];
            const double dx = pa.x - xi, dy = pa.y - yi, dz = pb.x - zi;
            const double s2 = fma(dz, dz, fma(dy, dy, dx * dx));
            const double y = rsqrt_seed(s2);
            const double e = fma(-s2, y * y, 1.0);
            const double rinv = fma(y, e * fma(0.375, e, 0.5), y);
            const double term = pb.y * rinv;
            acc += (jj >= jlo && s2 > 0.0) ? term : 0.0;
        }
    }
    double s = iok ? gm[i] * acc : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    if ((tid & 31) == 0) sh[tid >> 5] = s;
    __syncthreads();
    if (tid == 0) {
        double t = 0.0;
#pragma unroll
        for (int k = 0; k < EN_T / 32; ++k) t += sh[k];
        part[(size_t)blockIdx.y * gridDim.x + blockIdx.x] = t;
    }
}

// one block: partials -> out[7] = {G T, G Us, G Up, G E, G Lx, G Ly, G Lz} (gm units), fixed order
__global__ void __launch_bounds__(256) energy_final_kernel(const double* __restrict__ part_on, int n_on,
                                                           const double* __restrict__ part_pair, int n_pair, double mu,
                                                           double* __restrict__ out) {
    __shared__ double sh[256 / 32][EN_NSUM + 1];
    double s[EN_NSUM + 1];
#pragma unroll
    for (int k = 0; k <= EN_NSUM; ++k) s[k] = 0.0;
    for (int b = threadIdx.x; b < n_on; b += 256) {
#pragma unroll
        for (int k = 0; k < EN_NSUM; ++k) s[k] += part_on[(size_t)b * EN_NSUM + k];
    }
    for (int b = threadIdx.x; b < n_pair; b += 256) s[EN_NSUM] += part_pair[b];
#pragma unroll
    for (int k = 0; k <= EN_NSUM; ++k) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s[k] += __shfl_down_sync(0xffffffffu, s[k], o);
    }
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) {
#pragma unroll
        for (int k = 0; k <= EN_NSUM; ++k) sh[w][k] = s[k];
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double t[EN_NSUM + 1];
        for (int k = 0; k <= EN_NSUM; ++k) {
            t[k] = 0.0;
            for (int q = 0; q < 256 / 32; ++q) t[k] += sh[q][k];
        }
        // star: v_s = -P / mu  ->  1/2 mu v_s^2 = |P|^2 / (2 mu); its angular momentum cancels against
        // the barycentre shift of the bodies' positions (x_s cross (sum m v + m_star v_s) = 0)
        const double T = t[3] + 0.5 * (t[0] * t[0] + t[1] * t[1] + t[2] * t[2]) / mu;
        const double Us = -mu * t[4];
        const double Up = -t[EN_NSUM];
        out[0] = T; out[1] = Us; out[2] = Up; out[3] = T + Us + Up;
        out[4] = t[5]; out[5] = t[6]; out[6] = t[7];
    }
}

}  // namespace mopal
