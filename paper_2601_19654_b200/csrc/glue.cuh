// glue.cuh - the O(N) parts of the hybrid step (Hamiltonian block, and
// the drift loop), fused so that no per-body quantity goes through HBM more
// than once per stage (the whole step is 13 launches; step_small.cuh: 2 for small systems):
//   kick_psum_kernel        LOOP 1 (v += h/2 a)  + LOOP 2 partials (sum gm v)
//   jump_drift_boxes_kernel LOOP 2 finish + LOOP 3 (x += h/2 P/mu) + LOOP 4 (x0,v0 copy)
//                           + keplerian drift + mce_snif LOOP 1-2 (boxes) + the partials of
//                           sum gm v for the second jump
#pragma once
#include "common.cuh"
#include "encounters.cuh"
#include "kepler.cuh"
#include "pair_accel.cuh"

namespace mopal {

template <bool KICK>
__global__ void __launch_bounds__(ON_BLOCK) kick_psum_kernel(double* __restrict__ v, const double* __restrict__ a,
                                                              const double* __restrict__ gm, int nb, int ld,
                                                              double hk, double* psum, unsigned* ticket) {
    __shared__ double sh[ON_BLOCK / 32][3];
    const int b = blockIdx.x * ON_BLOCK + threadIdx.x;
    double s0 = 0, s1 = 0, s2 = 0;
    if (b < nb) {
        double vx = v[b], vy = v[ld + b], vz = v[2 * ld + b];
        if (KICK) {
            vx = fma(hk, a[b], vx); vy = fma(hk, a[ld + b], vy); vz = fma(hk, a[2 * ld + b], vz);
            v[b] = vx; v[ld + b] = vy; v[2 * ld + b] = vz;
        }
        const double g = gm[b];
        s0 = g * vx; s1 = g * vy; s2 = g * vz;
    }
    block_sum3<ON_BLOCK>(s0, s1, s2, sh);
    if (threadIdx.x == 0) { psum[3 * blockIdx.x] = s0; psum[3 * blockIdx.x + 1] = s1; psum[3 * blockIdx.x + 2] = s2; }
    psum_finalize<ON_BLOCK>(psum, gridDim.x, ticket, sh);
}

struct MidParams {
    double *x, *v, *x0, *v0;
    double *x1, *v1;        // nullable: second copy of the drifted state, read by the encounter pass while the
                            // jump / pair sum / kick branch already moves x and v (overlapped step)
    const double *gm, *rcrit;
    const double* psum_in;  // partials of sum gm v before the drift
    double* psum_out;       // partials after the drift
    unsigned* ticket;       // last-block counter of psum_out
    EncBuf enc;
    uint8_t* flag;
    DevStats* st;
    int nb, ld, nbPad, npsum, nbig;
    double hj_over_mu, mu, h;
};

__global__ void __launch_bounds__(ON_BLOCK) jump_drift_boxes_kernel(MidParams p) {
    __shared__ double sh[ON_BLOCK / 32][3];
    __shared__ float4 sh4[ON_BLOCK / 32];
    double P0, P1, P2;
    load_psum(p.psum_in, p.npsum, P0, P1, P2);
    const int b = blockIdx.x * ON_BLOCK + threadIdx.x;
    double s0 = 0, s1 = 0, s2 = 0;
    float4 bf = pad_boxf();
    if (b == 0) { *p.enc.nhit = 0ull; *p.enc.nlong = 0; }
    if (b < p.nbPad) { p.enc.rowcnt[b] = 0; p.enc.rowfill[b] = 0; }
    if (b < p.nb) {
        const int ld = p.ld;
        double x = p.x[b] + p.hj_over_mu * P0, y = p.x[ld + b] + p.hj_over_mu * P1, z = p.x[2 * ld + b] + p.hj_over_mu * P2;
        double vx = p.v[b], vy = p.v[ld + b], vz = p.v[2 * ld + b];
        p.x0[b] = x; p.x0[ld + b] = y; p.x0[2 * ld + b] = z;
        p.v0[b] = vx; p.v0[ld + b] = vy; p.v0[2 * ld + b] = vz;
        const double x0 = x, y0 = y, vx0 = vx, vy0 = vy;
        int iters;
        const int fail = drift_body(p.mu, p.h, x, y, z, vx, vy, vz, &iters);
        if (fail) atomicAdd(&p.st->drift_fail, 1);
        if (iters > 3) atomicMax(&p.st->max_newton, iters);
        p.x[b] = x; p.x[ld + b] = y; p.x[2 * ld + b] = z;
        p.v[b] = vx; p.v[ld + b] = vy; p.v[2 * ld + b] = vz;
        if (p.x1) {
            p.x1[b] = x; p.x1[ld + b] = y; p.x1[2 * ld + b] = z;
            p.v1[b] = vx; p.v1[ld + b] = vy; p.v1[2 * ld + b] = vz;
        }
        const double rc = b < p.nbig ? p.rcrit[b] : 0.0;   // LOOP 2 pads the big bodies only
        double lo, hi;
        double4 bx;
        box_1d(x0, x, vx0, vx, p.h, lo, hi);
        bx.x = __dsub_rn(lo, rc); bx.y = __dadd_rn(hi, rc);
        box_1d(y0, y, vy0, vy, p.h, lo, hi);
        bx.z = __dsub_rn(lo, rc); bx.w = __dadd_rn(hi, rc);
        p.enc.box[b] = bx;
        bf = box_f32(bx);
        p.enc.boxf[b] = bf;
        p.flag[b] = 0;
        const double g = p.gm[b];
        s0 = g * vx; s1 = g * vy; s2 = g * vz;
    } else if (b < p.nbPad) {
        p.enc.box[b] = pad_box();
        p.enc.boxf[b] = pad_boxf();
    }
    block_sum3<ON_BLOCK>(s0, s1, s2, sh);
    if (threadIdx.x == 0) { p.psum_out[3 * blockIdx.x] = s0; p.psum_out[3 * blockIdx.x + 1] = s1; p.psum_out[3 * blockIdx.x + 2] = s2; }
    psum_finalize<ON_BLOCK>(p.psum_out, p.npsum, p.ticket, sh);
    enc_bounds_partial(p.enc, b < p.nb, bf, sh4, p.nbPad / TJ);
}

// stand-alone drift (mo_drift)
__global__ void __launch_bounds__(ON_BLOCK, 4) drift_kernel(double* __restrict__ xx, double* __restrict__ vv, int nb, int ld,
                                                          double mu, double dt, DevStats* __restrict__ st) {
    const int b = blockIdx.x * ON_BLOCK + threadIdx.x;
    if (b >= nb) return;
    double x = xx[b], y = xx[ld + b], z = xx[2 * ld + b];
    double vx = vv[b], vy = vv[ld + b], vz = vv[2 * ld + b];
    int iters;
    const int fail = drift_body(mu, dt, x, y, z, vx, vy, vz, &iters);
    if (fail) atomicAdd(&st->drift_fail, 1);
    if (iters > 3) atomicMax(&st->max_newton, iters);
    xx[b] = x; xx[ld + b] = y; xx[2 * ld + b] = z;
    vv[b] = vx; vv[ld + b] = vy; vv[2 * ld + b] = vz;
}

__global__ void gm_kernel(const double* __restrict__ mass, double G, int nb, double* __restrict__ gm) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b < nb) gm[b] = G * mass[b];
}

// FP64 issue-peak probe: 8 independent DFMA chains per thread, register resident
__global__ void __launch_bounds__(256) dfma_probe_kernel(double* __restrict__ out, int iters, double b, double c) {
    double a0 = threadIdx.x, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
#pragma unroll 1
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            a0 = fma(a0, b, c); a1 = fma(a1, b, c); a2 = fma(a2, b, c); a3 = fma(a3, b, c);
            a4 = fma(a4, b, c); a5 = fma(a5, b, c); a6 = fma(a6, b, c); a7 = fma(a7, b, c);
        }
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
}

}  // namespace mopal
