/*
 * mopal_oracle.c - TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, obviously-correct CPU restatement of the hot path of Mercury's
 * hybrid symplectic step as the Mercury-Opal paper (arxiv 2601.19654) lays it
 * out: the O(N^2) K(r)-weighted mutual-gravity sum (force block, LOOP 2,
 * PAPER.md:150-165), the interaction/stellar-Hamiltonian block (kick, mvsum
 * reduction, jump, x0/v0 copy), the per-body Kepler drift
 * and the close-encounter check (mce_snif LOOPs 1-3,
 * PAPER.md:243-276), in the step order of PAPER.md:134.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / reference
 * legs may load this.  It shares no code, header, table or helper with the CUDA
 * path under paper_2601_19654_b200/csrc and neither includes the other.
 *
 * Arithmetic: every intermediate and every accumulator is `real`
 * (= long double, x87 80-bit, eps 5.4e-20) ; inputs and outputs are double.
 * Straight double loops in the paper's loop order, no tiling, no SIMD, no
 * reordering.  `#pragma omp parallel for` over the OUTER body loop only (each
 * body's own sum is still sequential, ascending j) - it changes no result.
 * Built a second time with -DORACLE_DOUBLE (real = double) purely as the timed
 * CPU baseline; the parity oracle is the long double build.
 *
 * The paper prints loop skeletons with the physics elided in <...> placeholders
 * and no equation; the arithmetic below follows the readings listed in
 * DESIGN.md section "Readings" (A-1..A-10, B-a..B-i, C-a..C-f, S-1..S-5), which
 * restate the paper's cited lineage (Chambers 1999; universal
 * variable Kepler solver as in WHFast).
 *
 * Layout: SoA planes, component c of body b at [c*ld + b], b = 0..nb-1
 * (paper index = b + 2; its element 1 is the star).
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"):
 *   accel      : mpmath brute force N<=8, Newton III, ring closed form, K limits,
 *                two-body closed form                               -> pinned
 *   boxes/pairs: mpmath brute force N<=8, straight-line closest approach closed
 *                form, dense sampling of the Hermite cubic, permutation /
 *                translation / time-reversal invariances            -> pinned
 *   drift      : period return + energy, circular closed form, fg determinant,
 *                group property, mpmath elements-based propagation  -> pinned
 *   step       : nb=1 by hand, angular momentum, reversibility, dt^2 energy
 *                scaling                                            -> pinned
 *   support    : h2dh/dh2h - mpmath centre of mass of the inertial N+1-body definition,
 *                two-body closed form, inverse; hill - exact cube closed form, Jupiter's
 *                textbook 0.355 AU, generator's a recovered by vis-viva, (1-e) ratio at
 *                perihelion; energy/L - two-body closed forms -GMm/2a and reduced-mass
 *                sqrt(mu a (1-e^2)), mpmath brute force over all N+1 bodies, dt^2
 *                scaling of the step's energy error                  -> pinned
 *   resolve    : no interaction left => the pinned Kepler drift; scipy DOP853 on the same
 *                equations written with the pinned changeover function (inside the shell, inside
 *                0.1 rc, negative h); time reversal; energy of the composed hybrid step through
 *                a close encounter with / without the encounter solve     -> pinned
 *   multi-step trajectories beyond ~10 steps: parity unpinned by construction
 *   (chaos; the paper itself compares curves and medians).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef ORACLE_DOUBLE
typedef double real;
#define R_SQRT sqrt
#define R_FABS fabs
#define R_EPS 2.220446049250313e-16
#else
typedef long double real;
#define R_SQRT sqrtl
#define R_FABS fabsl
#define R_EPS 1.0842021724855044e-19L
#endif

#define X_(p, c, b) ((real)(p)[(size_t)(c) * (size_t)ld + (size_t)(b)])

static inline real rmax(real a, real b) { return a > b ? a : b; }
static inline real rmin(real a, real b) { return a < b ? a : b; }

int oracle_real_bytes(void) { return (int)sizeof(real); }

/* Threads of the `omp parallel for` over the outer body loops (timing legs of bench.py: one thread
 * and all cores); n <= 0 only reports.  No arithmetic depends on it. */
#ifdef _OPENMP
#include <omp.h>
int oracle_set_num_threads(int n) { if (n > 0) omp_set_num_threads(n); return omp_get_max_threads(); }
#else
int oracle_set_num_threads(int n) { (void)n; return 1; }
#endif

/* ---------------------------------------------------------------------------
 * Changeover weight K(s ; rc)  [reading A-1, A-4, A-5; PAPER.md:104 fn. 14]
 *   q = (s - 0.1 rc) / (0.9 rc);  K = 0 (q<=0), 1 (q>=1), else q^3 (10 - 15 q + 6 q^2)
 * decided on squared quantities exactly as O-A states:
 *   s2 >= rc^2 -> 1 ; s2 <= (0.1 rc)^2 -> 0.
 * ------------------------------------------------------------------------- */
static real changeover_s2(real s2, real rc)
{
    real rc2 = rc * rc;
    if (s2 >= rc2) return 1;
    real rin = (real)0.1L * rc;
    if (s2 <= rin * rin) return 0;
    real s = R_SQRT(s2);
    real q = (s - rin) / ((real)0.9L * rc);
    return q * q * q * ((real)10 - (real)15 * q + (real)6 * q * q);
}

double oracle_changeover(double r, double rc)
{
    real rr = (real)r;
    return (double)changeover_s2(rr * rr, (real)rc);
}

/* ---------------------------------------------------------------------------
 * O-A  acceleration (force block LOOP 2):
 *   a_i = sum_{j != i} gm_j K_ij (x_j - x_i) / r_ij^3 ,  rc = max(rcrit_i, rcrit_j)
 * body-body terms only (the star is the drift's, the indirect term the jump's;
 * reading A-7).  S (nullable) receives sum_j |term| per component for the
 * parity tolerance |a_gpu - a_ref| <= 1e-12 S.
 * ------------------------------------------------------------------------- */
/* nsrc = number of gravity sources: the paper's inner loop runs over the big bodies only,
 * `do i = 2, nbig` inside `do j = 2, nbod` ("only the massive ones, labeled
 * as big bodies in the software, are also gravity sources").  Sources are bodies
 * 0..nsrc-1; nsrc = nb is the fully interacting case (reading R-1). */
static void accel_row(int nb, int nsrc, int ld, const double *gm, const double *x, const double *rcrit,
                      int i, real *acc3, real *abs3)
{
    (void)nb;
    real xi = X_(x, 0, i), yi = X_(x, 1, i), zi = X_(x, 2, i);
    real rci = (real)rcrit[i];
    real ax = 0, ay = 0, az = 0, sx = 0, sy = 0, sz = 0;
    for (int j = 0; j < nsrc; ++j) {
        if (j == i) continue;
        real dx = X_(x, 0, j) - xi;
        real dy = X_(x, 1, j) - yi;
        real dz = X_(x, 2, j) - zi;
        real s2 = dx * dx + dy * dy + dz * dz;
        if (s2 == 0) continue;                       /* reading A-9 */
        real rc = rmax(rci, (real)rcrit[j]);         /* reading A-3 */
        real K = changeover_s2(s2, rc);
        if (K == 0) continue;
        real w = (real)gm[j] * K / (s2 * R_SQRT(s2));
        ax += w * dx; ay += w * dy; az += w * dz;
        sx += R_FABS(w * dx); sy += R_FABS(w * dy); sz += R_FABS(w * dz);
    }
    acc3[0] = ax; acc3[1] = ay; acc3[2] = az;
    abs3[0] = sx; abs3[1] = sy; abs3[2] = sz;
}

int oracle_accel_big(int nb, int nbig, int ld, const double *gm, const double *x,
                     const double *rcrit, double *a, double *S)
{
    if (nb < 0 || ld < nb || nbig < 0 || nbig > nb) return 1;
#pragma omp parallel for schedule(static)
    for (int i = 0; i < nb; ++i) {
        real acc[3], ab[3];
        accel_row(nb, nbig, ld, gm, x, rcrit, i, acc, ab);
        for (int c = 0; c < 3; ++c) {
            a[(size_t)c * ld + i] = (double)acc[c];
            if (S) S[(size_t)c * ld + i] = (double)ab[c];
        }
    }
    return 0;
}

int oracle_accel(int nb, int ld, const double *gm, const double *x,
                 const double *rcrit, double *a, double *S)
{
    return oracle_accel_big(nb, nb, ld, gm, x, rcrit, a, S);
}

/* the same sum for a chosen subset of bodies i (full-size sampled parity):
 * a_out / S_out are [3][nrows]. */
int oracle_accel_rows_big(int nb, int nbig, int ld, const double *gm, const double *x, const double *rcrit,
                          const int32_t *rows, int nrows, double *a_out, double *S_out)
{
    if (nb < 0 || ld < nb || nrows < 0 || nbig < 0 || nbig > nb) return 1;
#pragma omp parallel for schedule(dynamic, 1)
    for (int k = 0; k < nrows; ++k) {
        real acc[3], ab[3];
        if (rows[k] < 0 || rows[k] >= nb) continue;
        accel_row(nb, nbig, ld, gm, x, rcrit, rows[k], acc, ab);
        for (int c = 0; c < 3; ++c) {
            a_out[(size_t)c * nrows + k] = (double)acc[c];
            if (S_out) S_out[(size_t)c * nrows + k] = (double)ab[c];
        }
    }
    return 0;
}

int oracle_accel_rows(int nb, int ld, const double *gm, const double *x, const double *rcrit,
                      const int32_t *rows, int nrows, double *a_out, double *S_out)
{
    return oracle_accel_rows_big(nb, nb, ld, gm, x, rcrit, rows, nrows, a_out, S_out);
}

/* ---------------------------------------------------------------------------
 * O-B.1  boxes (mce_snif LOOP 1 + LOOP 2; readings B-a,b,c)
 * Per body and per coordinate c in {x, y}: extremes of the cubic Hermite
 * interpolant through (p0, h w0) at tau=0 and (p1, h w1) at tau=1, padded by
 * rcrit.  lo/hi: [2][nb] (x plane then y plane).
 * ------------------------------------------------------------------------- */
static void box_1d(real p0, real p1, real w0, real w1, real h, real *lo, real *hi)
{
    real l = rmin(p0, p1), u = rmax(p0, p1);
    if (w0 * w1 < 0) {
        real k1 = h * w0;
        real k2 = -(real)3 * p0 - (real)2 * h * w0 + (real)3 * p1 - h * w1;
        real k3 = (real)2 * p0 + h * w0 - (real)2 * p1 + h * w1;
        real D = k2 * k2 - (real)3 * k3 * k1;
        if (D >= 0) {
            real sq = R_SQRT(D);
            real qq = (k2 >= 0) ? (k2 + sq) : (k2 - sq);
            if (qq != 0) {
                real ta = -k1 / qq;
                if (ta > 0 && ta < 1) {
                    real p = ((k3 * ta + k2) * ta + k1) * ta + p0;
                    l = rmin(l, p); u = rmax(u, p);
                }
            }
            if (k3 != 0) {
                real tb = -qq / ((real)3 * k3);
                if (tb > 0 && tb < 1) {
                    real p = ((k3 * tb + k2) * tb + k1) * tb + p0;
                    l = rmin(l, p); u = rmax(u, p);
                }
            }
        }
    }
    *lo = l; *hi = u;
}

/* nbig: LOOP 2 adds rcrit to the extremes of the big bodies only, `do j = 2, nbig`
 * (PAPER.md:249-253); nbig = nb pads every box (reading B-c; R-2). */
static void boxes_real(int nb, int nbig, int ld, real h, const double *x0, const double *v0,
                       const double *x1, const double *v1, const double *rcrit,
                       real *lo, real *hi)
{
#pragma omp parallel for schedule(static)
    for (int b = 0; b < nb; ++b) {
        for (int c = 0; c < 2; ++c) {
            real l, u;
            box_1d(X_(x0, c, b), X_(x1, c, b), X_(v0, c, b), X_(v1, c, b), h, &l, &u);
            real pad = (b < nbig) ? (real)rcrit[b] : (real)0;
            lo[(size_t)c * nb + b] = l - pad;
            hi[(size_t)c * nb + b] = u + pad;
        }
    }
}

int oracle_boxes_big(int nb, int nbig, int ld, double h, const double *x0, const double *v0,
                     const double *x1, const double *v1, const double *rcrit,
                     double *lo, double *hi)
{
    if (nb < 0 || ld < nb || nbig < 0 || nbig > nb) return 1;
    real *l = (real *)malloc(sizeof(real) * 2 * (size_t)(nb + 1));
    real *u = (real *)malloc(sizeof(real) * 2 * (size_t)(nb + 1));
    if (!l || !u) { free(l); free(u); return 2; }
    boxes_real(nb, nbig, ld, (real)h, x0, v0, x1, v1, rcrit, l, u);
    for (size_t k = 0; k < 2 * (size_t)nb; ++k) { lo[k] = (double)l[k]; hi[k] = (double)u[k]; }
    free(l); free(u);
    return 0;
}

int oracle_boxes(int nb, int ld, double h, const double *x0, const double *v0,
                 const double *x1, const double *v1, const double *rcrit,
                 double *lo, double *hi)
{
    return oracle_boxes_big(nb, nb, ld, h, x0, v0, x1, v1, rcrit, lo, hi);
}

/* ---------------------------------------------------------------------------
 * O-B.2  minimum separation estimate of one pair over the step (mce_min,
 * PAPER.md:261-262, 281-283; reading B-d): cubic Hermite interpolant of the
 * SQUARED separation, interior minimum only when approaching at the start and
 * receding at the end.  Returns d2min; d0/d1 (nullable) get the end values.
 * ------------------------------------------------------------------------- */
static real pair_d2min(int ld, real h, const double *x0, const double *v0,
                       const double *x1, const double *v1, int i, int j,
                       real *d0_out, real *d1_out)
{
    real d0 = 0, d1 = 0, s0 = 0, s1 = 0;
    for (int c = 0; c < 3; ++c) {
        real D0 = X_(x0, c, i) - X_(x0, c, j);
        real D1 = X_(x1, c, i) - X_(x1, c, j);
        real U0 = X_(v0, c, i) - X_(v0, c, j);
        real U1 = X_(v1, c, i) - X_(v1, c, j);
        d0 += D0 * D0; d1 += D1 * D1;
        s0 += D0 * U0; s1 += D1 * U1;
    }
    real d0t = (real)2 * s0, d1t = (real)2 * s1;
    real d2min;
    if (d0t * h <= 0 && d1t * h >= 0) {
        real c1 = h * d0t;
        real c2 = -(real)3 * d0 - (real)2 * h * d0t + (real)3 * d1 - h * d1t;
        real c3 = (real)2 * d0 + h * d0t - (real)2 * d1 + h * d1t;
        real D = rmax(c2 * c2 - (real)3 * c3 * c1, 0);
        real den = c2 + R_SQRT(D);
        real tau = (den > 0) ? (-c1 / den) : (real)0;
        tau = rmin(rmax(tau, 0), 1);
        d2min = rmax(((c3 * tau + c2) * tau + c1) * tau + d0, 0);
        d2min = rmin(d2min, rmin(d0, d1));
    } else {
        d2min = rmin(d0, d1);
    }
    if (d0_out) *d0_out = d0;
    if (d1_out) *d1_out = d1;
    return d2min;
}

double oracle_pair_d2min(int ld, double h, const double *x0, const double *v0,
                         const double *x1, const double *v1, int i, int j)
{
    return (double)pair_d2min(ld, (real)h, x0, v0, x1, v1, i, j, 0, 0);
}

/* classify one pair: 0 = out, 1 = in (flagged), bit 1 set (|2) = ambiguous:
 * some comparison deciding the outcome sits within 1e-12 relative of equality
 * (north_star: lists bit-exact "except for pairs within 1e-12 relative of a
 * threshold"). */
#define AMBIG_TOL ((real)1e-12L)
static int near_eq(real a, real b, real scale)
{
    return R_FABS(a - b) <= AMBIG_TOL * scale;
}

static int classify_pair(int nb, int ld, real h, const double *x0, const double *v0,
                         const double *x1, const double *v1, const double *rcrit,
                         const real *lo, const real *hi, int i, int j)
{
    int amb = 0, gate = 1;
    for (int c = 0; c < 2; ++c) {                        /* box gate, reading B-f */
        real li = lo[(size_t)c * nb + i], ui = hi[(size_t)c * nb + i];
        real lj = lo[(size_t)c * nb + j], uj = hi[(size_t)c * nb + j];
        if (!(li <= uj)) gate = 0;
        if (!(lj <= ui)) gate = 0;
        if (near_eq(li, uj, rmax(R_FABS(li), R_FABS(uj)))) amb = 1;
        if (near_eq(lj, ui, rmax(R_FABS(lj), R_FABS(ui)))) amb = 1;
    }
    if (!gate && !amb) return 0;
    real d0, d1;
    real d2 = pair_d2min(ld, h, x0, v0, x1, v1, i, j, &d0, &d1);
    real rc = rmax((real)rcrit[i], (real)rcrit[j]);      /* reading B-e */
    real rc2 = rc * rc;
    int in = gate && (d2 <= rc2);
    int amb2 = near_eq(d2, rc2, rmax(rc2, rmax(d0, d1)));
    /* ambiguity matters only if flipping the near-equal comparison could flip
       the outcome: a near-equal gate with the distance test failing clearly is
       still a clear "out". */
    int ambiguous = 0;
    if (amb2 && (gate || amb)) ambiguous = 1;
    if (amb && (d2 <= rc2 || amb2)) ambiguous = 1;
    return in | (ambiguous ? 2 : 0);
}

/* ---------------------------------------------------------------------------
 * O-B  encounter list (mce_snif LOOP 3).  All i<j, ascending
 * i then ascending j (the paper's order is whatever its atomics give,
 * PAPER.md:264-269; reading B-g).  pairs: 2*cap int32 (i,j interleaved), count
 * returned is the TRUE total even if > cap.  flag[b]=1 iff b is in a flagged
 * pair (paper: ce=2).  ambig (nullable): pairs whose outcome
 * is within 1e-12 relative of a threshold, n_ambig = their true number.
 * ------------------------------------------------------------------------- */
/* nbig: LOOP 3 runs `do i = 2, nbig` x `do j = 2, nbod`, j > i: the first
 * body of a pair is a big body; nbig = nb tests every pair (reading R-3). */
static int64_t encounters_impl(int nb, int nbig, int ld, double h_, const double *x0, const double *v0,
                               const double *x1, const double *v1, const double *rcrit,
                               int32_t *pairs, int64_t cap, uint8_t *flag,
                               int32_t *ambig, int64_t ambig_cap, int64_t *n_ambig,
                               int row_stride, int row_phase)
{
    if (nb < 0 || ld < nb || nbig < 0 || nbig > nb) return -1;
    real h = (real)h_;
    real *lo = (real *)malloc(sizeof(real) * 2 * (size_t)(nb + 1));
    real *hi = (real *)malloc(sizeof(real) * 2 * (size_t)(nb + 1));
    int64_t *rowcnt = (int64_t *)calloc((size_t)nb + 1, sizeof(int64_t));
    int64_t *rowamb = (int64_t *)calloc((size_t)nb + 1, sizeof(int64_t));
    if (!lo || !hi || !rowcnt || !rowamb) { free(lo); free(hi); free(rowcnt); free(rowamb); return -2; }
    boxes_real(nb, nbig, ld, h, x0, v0, x1, v1, rcrit, lo, hi);
    if (flag) memset(flag, 0, (size_t)nb);
    /* pass 1: per-row counts */
#pragma omp parallel for schedule(dynamic, 16)
    for (int i = 0; i < nbig; ++i) {
        int64_t c = 0, ca = 0;
        if (i % row_stride != row_phase) continue;
        for (int j = i + 1; j < nb; ++j) {
            int r = classify_pair(nb, ld, h, x0, v0, x1, v1, rcrit, lo, hi, i, j);
            c += (r & 1); ca += ((r >> 1) & 1);
        }
        rowcnt[i] = c; rowamb[i] = ca;
    }
    int64_t total = 0, total_a = 0;
    for (int i = 0; i < nb; ++i) {
        int64_t c = rowcnt[i], ca = rowamb[i];
        rowcnt[i] = total; rowamb[i] = total_a;
        total += c; total_a += ca;
    }
    /* pass 2: fill in order */
#pragma omp parallel for schedule(dynamic, 16)
    for (int i = 0; i < nbig; ++i) {
        int64_t o = rowcnt[i], oa = rowamb[i];
        int64_t ne = ((i + 1 < nb) ? rowcnt[i + 1] : total) - o;
        int64_t na = ((i + 1 < nb) ? rowamb[i + 1] : total_a) - oa;
        if (ne == 0 && na == 0) continue;
        for (int j = i + 1; j < nb; ++j) {
            int r = classify_pair(nb, ld, h, x0, v0, x1, v1, rcrit, lo, hi, i, j);
            if (r & 1) {
                if (pairs && o < cap) { pairs[2 * o] = i; pairs[2 * o + 1] = j; }
                ++o;
                if (flag) {                              /* from the definition, not the (maybe truncated) list */
#pragma omp atomic write
                    flag[i] = 1;
#pragma omp atomic write
                    flag[j] = 1;
                }
            }
            if (r & 2) {
                if (ambig && oa < ambig_cap) { ambig[2 * oa] = i; ambig[2 * oa + 1] = j; }
                ++oa;
            }
        }
    }
    if (n_ambig) *n_ambig = total_a;
    free(lo); free(hi); free(rowcnt); free(rowamb);
    return total;
}

int64_t oracle_encounters(int nb, int ld, double h_, const double *x0, const double *v0,
                          const double *x1, const double *v1, const double *rcrit,
                          int32_t *pairs, int64_t cap, uint8_t *flag,
                          int32_t *ambig, int64_t ambig_cap, int64_t *n_ambig)
{
    return encounters_impl(nb, nb, ld, h_, x0, v0, x1, v1, rcrit, pairs, cap, flag, ambig, ambig_cap,
                           n_ambig, 1, 0);
}

/* the same list restricted to rows i with i % row_stride == row_phase (full-size sampled
 * parity); flag then marks only bodies of those pairs. */
int64_t oracle_encounters_rows(int nb, int ld, double h_, const double *x0, const double *v0,
                               const double *x1, const double *v1, const double *rcrit,
                               int32_t *pairs, int64_t cap, uint8_t *flag,
                               int32_t *ambig, int64_t ambig_cap, int64_t *n_ambig,
                               int row_stride, int row_phase)
{
    if (row_stride < 1 || row_phase < 0 || row_phase >= row_stride) return -1;
    return encounters_impl(nb, nb, ld, h_, x0, v0, x1, v1, rcrit, pairs, cap, flag, ambig, ambig_cap,
                           n_ambig, row_stride, row_phase);
}

int64_t oracle_encounters_big(int nb, int nbig, int ld, double h_, const double *x0, const double *v0,
                              const double *x1, const double *v1, const double *rcrit,
                              int32_t *pairs, int64_t cap, uint8_t *flag,
                              int32_t *ambig, int64_t ambig_cap, int64_t *n_ambig,
                              int row_stride, int row_phase)
{
    if (row_stride < 1 || row_phase < 0 || row_phase >= row_stride) return -1;
    return encounters_impl(nb, nbig, ld, h_, x0, v0, x1, v1, rcrit, pairs, cap, flag, ambig, ambig_cap,
                           n_ambig, row_stride, row_phase);
}

/* ---------------------------------------------------------------------------
 * O-C  Kepler drift (arxes_drift; readings C-a..C-f).
 * Universal variables: c_n(z) = sum_k (-z)^k / (2k+n)!,  G_n = X^n c_n(beta X^2)
 *   solve  r0 G1 + eta0 G2 + mu G3 = dt  for X   (F' = r > 0: unique root)
 *   f = 1 - mu G2 / r0, g = dt - mu G3, fdot = -mu G1 / (r0 r), gdot = 1 - mu G2 / r
 * ------------------------------------------------------------------------- */
static void stumpff(real z, real *c0, real *c1, real *c2, real *c3)
{
    int n = 0;
    while (R_FABS(z) > (real)0.1L) { z *= (real)0.25L; ++n; }
    /* series: c2 = 1/2! - z/4! + z^2/6! - ... ; c3 = 1/3! - z/5! + z^2/7! - ... */
    real t2 = (real)0.5L, t3 = (real)1 / (real)6, s2 = 0, s3 = 0;
    for (int k = 1; k <= 30; ++k) {
        s2 += t2; s3 += t3;
        t2 *= -z / (real)((2 * k + 1) * (2 * k + 2));
        t3 *= -z / (real)((2 * k + 2) * (2 * k + 3));
        if (R_FABS(t2) < R_EPS * (real)0.01L && R_FABS(t3) < R_EPS * (real)0.01L) break;
    }
    s2 += t2; s3 += t3;
    real C2 = s2, C3 = s3;
    real C1 = (real)1 - z * C3;
    real C0 = (real)1 - z * C2;
    for (; n > 0; --n) {                                 /* undo each quartering */
        C3 = (C2 + C0 * C3) * (real)0.25L;
        C2 = C1 * C1 * (real)0.5L;
        C1 = C0 * C1;
        C0 = (real)2 * C0 * C0 - (real)1;
    }
    *c0 = C0; *c1 = C1; *c2 = C2; *c3 = C3;
}

static void gfuncs(real X, real beta, real *G0, real *G1, real *G2, real *G3)
{
    real c0, c1, c2, c3;
    real X2 = X * X;
    stumpff(beta * X2, &c0, &c1, &c2, &c3);
    *G0 = c0; *G1 = X * c1; *G2 = X2 * c2; *G3 = X2 * X * c3;
}

/* one body; returns 0 ok, 1 failed (state untouched) */
static int drift_one(real mu, real dt, real *px, real *pv)
{
    real x0 = px[0], y0 = px[1], z0 = px[2], vx = pv[0], vy = pv[1], vz = pv[2];
    real r0 = R_SQRT(x0 * x0 + y0 * y0 + z0 * z0);
    if (!(r0 > 0)) return 1;                             /* reading C-f */
    real v2 = vx * vx + vy * vy + vz * vz;
    real eta0 = x0 * vx + y0 * vy + z0 * vz;
    real beta = (real)2 * mu / r0 - v2;
    real X = dt / r0, G0, G1, G2, G3, r = r0;
    int conv = 0;
    for (int it = 0; it < 60; ++it) {
        gfuncs(X, beta, &G0, &G1, &G2, &G3);
        real F = r0 * G1 + eta0 * G2 + mu * G3 - dt;
        r = r0 * G0 + eta0 * G1 + mu * G2;
        if (!(r > 0) || !isfinite((double)F)) break;
        real dX = -F / r;
        X += dX;
        if (R_FABS(dX) <= (real)4 * R_EPS * R_FABS(X)) { conv = 1; break; }
    }
    if (!conv) {
        /* bisection on a bracket grown from 0 (F(0) = -dt, F monotone in X) */
        real sgn = dt >= 0 ? (real)1 : (real)-1;
        real a = 0, b = sgn * R_FABS(dt / r0);
        int ok = 0;
        for (int it = 0; it < 200; ++it) {
            gfuncs(b, beta, &G0, &G1, &G2, &G3);
            real F = r0 * G1 + eta0 * G2 + mu * G3 - dt;
            if (!isfinite((double)F)) return 1;
            if (F * sgn >= 0) { ok = 1; break; }
            a = b; b *= (real)2;
        }
        if (!ok) return 1;
        for (int it = 0; it < 200; ++it) {
            real m = (real)0.5L * (a + b);
            gfuncs(m, beta, &G0, &G1, &G2, &G3);
            real F = r0 * G1 + eta0 * G2 + mu * G3 - dt;
            if (F * sgn >= 0) b = m; else a = m;
            if (R_FABS(b - a) <= (real)2 * R_EPS * R_FABS(b)) break;
        }
        X = (real)0.5L * (a + b);
    }
    gfuncs(X, beta, &G0, &G1, &G2, &G3);
    r = r0 * G0 + eta0 * G1 + mu * G2;
    if (!(r > 0)) return 1;
    real fm1 = -mu * G2 / r0;                            /* f - 1 */
    real g = dt - mu * G3;
    real fd = -mu * G1 / (r0 * r);
    real gdm1 = -mu * G2 / r;                            /* gdot - 1 */
    px[0] = x0 + (fm1 * x0 + g * vx);
    px[1] = y0 + (fm1 * y0 + g * vy);
    px[2] = z0 + (fm1 * z0 + g * vz);
    pv[0] = vx + (fd * x0 + gdm1 * vx);
    pv[1] = vy + (fd * y0 + gdm1 * vy);
    pv[2] = vz + (fd * z0 + gdm1 * vz);
    return 0;
}

/* x, v in place; iflag (nullable) per body: 0 ok, 1 failed.  Returns #failed. */
int oracle_drift(int nb, int ld, double mu, double dt, double *x, double *v, int32_t *iflag)
{
    if (nb < 0 || ld < nb) return -1;
    int nfail = 0;
#pragma omp parallel for schedule(static) reduction(+ : nfail)
    for (int b = 0; b < nb; ++b) {
        real px[3], pv[3];
        for (int c = 0; c < 3; ++c) { px[c] = X_(x, c, b); pv[c] = X_(v, c, b); }
        int f = drift_one((real)mu, (real)dt, px, pv);
        if (!f) {
            for (int c = 0; c < 3; ++c) {
                x[(size_t)c * ld + b] = (double)px[c];
                v[(size_t)c * ld + b] = (double)pv[c];
            }
        }
        if (iflag) iflag[b] = f;
        nfail += f;
    }
    return nfail;
}

/* ---------------------------------------------------------------------------
 * Hamiltonian block pieces
 * ------------------------------------------------------------------------- */
/* LOOP 1: v_j += hk a_j */
int oracle_kick(int nb, int ld, double hk, double *v, const double *a)
{
#pragma omp parallel for schedule(static)
    for (int b = 0; b < nb; ++b)
        for (int c = 0; c < 3; ++c)
            v[(size_t)c * ld + b] = (double)(X_(v, c, b) + (real)hk * X_(a, c, b));
    return 0;
}

/* LOOP 2: mvsum = sum_j gm_j v_j (ascending j) ; LOOP 3: x_j += hj mvsum / mu */
int oracle_jump(int nb, int ld, double hj, double mu, const double *gm, double *x,
                const double *v, double *P3)
{
    real P[3] = {0, 0, 0};
    for (int b = 0; b < nb; ++b)
        for (int c = 0; c < 3; ++c) P[c] += (real)gm[b] * X_(v, c, b);
#pragma omp parallel for schedule(static)
    for (int b = 0; b < nb; ++b)
        for (int c = 0; c < 3; ++c)
            x[(size_t)c * ld + b] = (double)(X_(x, c, b) + (real)hj * P[c] / (real)mu);
    if (P3) for (int c = 0; c < 3; ++c) P3[c] = (double)P[c];
    return 0;
}

/* ---------------------------------------------------------------------------
 * O-D  one hybrid step of size h (mdt_hy, Fig. 1; readings S-1..S-5):
 *   kick h/2 -> jump h/2 -> copy x0,v0 -> drift h -> encounter check ->
 *   jump h/2 (mvsum from the drifted v) -> a = accel(x) -> kick h/2.
 * `a` must be current for `x` on entry; it is current for the new x on exit.
 * No restore and no encounter resolution (reading S-3).  nbig < nb: the force sum and the
 * encounter check use the big bodies as sources / first members (R-1..R-3); kick, mvsum, jump,
 * copy and drift run over all bodies, `do j = 2, nbod`.
 * Returns the encounter count of this step (<0 on error); *nfail = drift failures.
 * ------------------------------------------------------------------------- */
int64_t oracle_step_big(int nb, int nbig, int ld, double mu, const double *gm, const double *rcrit,
                    double h, double *x, double *v, double *a, double *x0, double *v0,
                    int32_t *pairs, int64_t cap, uint8_t *flag,
                    int32_t *ambig, int64_t ambig_cap, int64_t *n_ambig, int32_t *nfail)
{
    if (nb < 0 || ld < nb || nbig < 0 || nbig > nb) return -1;
    oracle_kick(nb, ld, 0.5 * h, v, a);
    oracle_jump(nb, ld, 0.5 * h, mu, gm, x, v, 0);
    for (int c = 0; c < 3; ++c) {                        /* LOOP 4 */
        memcpy(x0 + (size_t)c * ld, x + (size_t)c * ld, sizeof(double) * (size_t)nb);
        memcpy(v0 + (size_t)c * ld, v + (size_t)c * ld, sizeof(double) * (size_t)nb);
    }
    int nf = oracle_drift(nb, ld, mu, h, x, v, 0);
    if (nfail) *nfail = nf;
    int64_t cnt = oracle_encounters_big(nb, nbig, ld, h, x0, v0, x, v, rcrit, pairs, cap, flag,
                                        ambig, ambig_cap, n_ambig, 1, 0);
    oracle_jump(nb, ld, 0.5 * h, mu, gm, x, v, 0);
    oracle_accel_big(nb, nbig, ld, gm, x, rcrit, a, 0);
    oracle_kick(nb, ld, 0.5 * h, v, a);
    return cnt;
}

int64_t oracle_step(int nb, int ld, double mu, const double *gm, const double *rcrit,
                    double h, double *x, double *v, double *a, double *x0, double *v0,
                    int32_t *pairs, int64_t cap, uint8_t *flag,
                    int32_t *ambig, int64_t ambig_cap, int64_t *n_ambig, int32_t *nfail)
{
    return oracle_step_big(nb, nb, ld, mu, gm, rcrit, h, x, v, a, x0, v0, pairs, cap, flag,
                           ambig, ambig_cap, n_ambig, nfail);
}

/* step without the O(N^2/2) encounter pass, for long multi-step invariant pins */
int oracle_step_noenc(int nb, int ld, double mu, const double *gm, const double *rcrit,
                      double h, double *x, double *v, double *a)
{
    if (nb < 0 || ld < nb) return -1;
    oracle_kick(nb, ld, 0.5 * h, v, a);
    oracle_jump(nb, ld, 0.5 * h, mu, gm, x, v, 0);
    oracle_drift(nb, ld, mu, h, x, v, 0);
    oracle_jump(nb, ld, 0.5 * h, mu, gm, x, v, 0);
    oracle_accel(nb, ld, gm, x, rcrit, a, 0);
    oracle_kick(nb, ld, 0.5 * h, v, a);
    return 0;
}

/* ---------------------------------------------------------------------------
 * Per-step support routines the paper names next to the hot path:
 * coordinate conversion heliocentric <-> democratic heliocentric (mco_h2dh, mce_dh2h;
 * PAPER.md:84 item 1 and fn. 12), Hill and critical radii (mce_hill, mce_init;
 * PAPER.md:87, 94, fn. 14, and 291 item 3: "critical radii are always updated since they
 * depend on the instantaneous distance between each planet and the central star"), total
 * energy and momentum (mxx_en).  The paper states what they compute in words
 * only; the arithmetic follows readings H-1..H-4 and E-1..E-3.
 * Masses in Msun (not gm): these routines need mass ratios and G separately.
 * ------------------------------------------------------------------------- */
#ifdef ORACLE_DOUBLE
#define R_CBRT cbrt
#else
#define R_CBRT cbrtl
#endif

/* sum_k m_k v_k, ascending k */
static void mv_sum(int nb, int ld, const double *mass, const double *v, real S[3])
{
    S[0] = S[1] = S[2] = 0;
    for (int b = 0; b < nb; ++b)
        for (int c = 0; c < 3; ++c) S[c] += (real)mass[b] * X_(v, c, b);
}

/* H-1: heliocentric -> democratic heliocentric.  Positions stay heliocentric; velocities
 * become barycentric: v_j -= sum_k m_k v_k / (mstar + sum_k m_k)  (the star's heliocentric
 * velocity is 0, so the barycentre moves at sum m v / M_total in the heliocentric frame). */
int oracle_h2dh(int nb, int ld, double mstar, const double *mass, double *v)
{
    if (nb < 0 || ld < nb) return -1;
    real S[3], mtot = (real)mstar;
    mv_sum(nb, ld, mass, v, S);
    for (int b = 0; b < nb; ++b) mtot += (real)mass[b];
    for (int b = 0; b < nb; ++b)
        for (int c = 0; c < 3; ++c)
            v[(size_t)c * ld + b] = (double)(X_(v, c, b) - S[c] / mtot);
    return 0;
}

/* H-2: democratic heliocentric -> heliocentric: v_j += sum_k m_k v_k / mstar
 * (barycentric momentum is zero, so the star moves at -sum m v / mstar). */
int oracle_dh2h(int nb, int ld, double mstar, const double *mass, double *v)
{
    if (nb < 0 || ld < nb) return -1;
    real S[3];
    mv_sum(nb, ld, mass, v, S);
    for (int b = 0; b < nb; ++b)
        for (int c = 0; c < 3; ++c)
            v[(size_t)c * ld + b] = (double)(X_(v, c, b) + S[c] / (real)mstar);
    return 0;
}

/* H-3 / H-4: Hill radius r_H = d (m / 3 mstar)^(1/3) and critical radius rcrit = nhill r_H.
 * mode 0 (default reading of PAPER.md:94, 291): d = |x_j|, the instantaneous star-planet separation.
 * mode 1 (variant): d = osculating semi-major axis, 1/a = 2/r - v_h^2 / (G (mstar + m_j)), with the
 *        heliocentric velocity v_h = v + sum m v / mstar of the democratic heliocentric input (H-2);
 *        unbound bodies (1/a <= 0) fall back to d = r.
 * x heliocentric, v barycentric (democratic heliocentric), as everywhere on the path. */
int oracle_hill(int nb, int ld, int mode, double nhill, double G, double mstar, const double *mass,
                const double *x, const double *v, double *rhill, double *rcrit)
{
    if (nb < 0 || ld < nb || (mode != 0 && mode != 1)) return -1;
    real S[3] = {0, 0, 0};
    if (mode == 1) mv_sum(nb, ld, mass, v, S);
#pragma omp parallel for schedule(static)
    for (int b = 0; b < nb; ++b) {
        real r2 = 0;
        for (int c = 0; c < 3; ++c) r2 += X_(x, c, b) * X_(x, c, b);
        real d = R_SQRT(r2);
        if (mode == 1) {
            real v2 = 0;
            for (int c = 0; c < 3; ++c) {
                real vh = X_(v, c, b) + S[c] / (real)mstar;
                v2 += vh * vh;
            }
            real inva = (real)2 / d - v2 / ((real)G * ((real)mstar + (real)mass[b]));
            if (inva > 0) d = (real)1 / inva;
        }
        real rh = d * R_CBRT((real)mass[b] / ((real)3 * (real)mstar));
        if (rhill) rhill[b] = (double)rh;
        if (rcrit) rcrit[b] = (double)((real)nhill * rh);
    }
    return 0;
}

/* E-1..E-3: total energy and angular momentum of star + bodies in the barycentric frame, from
 * democratic heliocentric input (x heliocentric, v barycentric):
 *   star:  v_s = -sum m v / mstar,  x_s = -sum m x / (mstar + sum m)   (barycentric)
 *   T  = 1/2 sum m v^2 + 1/2 mstar v_s^2
 *   Us = -G mstar sum m_j / |x_j|
 *   Up = -G sum_{i<j, i<nbig} m_i m_j / |x_i - x_j|     (the pairs that interact: first member big,
 *                                                        PAPER.md:152-157; nbig = nb: all pairs)
 *   L  = sum m (x + x_s) x v + mstar x_s x v_s
 * out[0..10] = T, Us, Up, E = T+Us+Up, Lx, Ly, Lz, sum|energy terms|, sum|L terms| per component. */
int oracle_energy(int nb, int nbig, int ld, double G, double mstar, const double *mass,
                  const double *x, const double *v, double *out)
{
    if (nb < 0 || ld < nb || nbig < 0 || nbig > nb) return -1;
    real Sv[3], Sx[3] = {0, 0, 0}, mtot = (real)mstar;
    mv_sum(nb, ld, mass, v, Sv);
    for (int b = 0; b < nb; ++b) {
        mtot += (real)mass[b];
        for (int c = 0; c < 3; ++c) Sx[c] += (real)mass[b] * X_(x, c, b);
    }
    real xs[3], vs[3];
    for (int c = 0; c < 3; ++c) { xs[c] = -Sx[c] / mtot; vs[c] = -Sv[c] / (real)mstar; }
    real T = 0, Us = 0, Eabs = 0, L[3] = {0, 0, 0}, Labs[3] = {0, 0, 0};
    for (int b = 0; b < nb; ++b) {
        real m = (real)mass[b], r2 = 0, v2 = 0, p[3], w[3];
        for (int c = 0; c < 3; ++c) {
            p[c] = X_(x, c, b) + xs[c]; w[c] = X_(v, c, b);
            r2 += X_(x, c, b) * X_(x, c, b); v2 += w[c] * w[c];
        }
        T += (real)0.5L * m * v2;
        real us = (real)G * (real)mstar * m / R_SQRT(r2);
        Us -= us;
        Eabs += (real)0.5L * m * v2 + us;
        real l[3] = {p[1] * w[2] - p[2] * w[1], p[2] * w[0] - p[0] * w[2], p[0] * w[1] - p[1] * w[0]};
        for (int c = 0; c < 3; ++c) { L[c] += m * l[c]; Labs[c] += R_FABS(m * l[c]); }
    }
    {
        real v2 = vs[0] * vs[0] + vs[1] * vs[1] + vs[2] * vs[2];
        T += (real)0.5L * (real)mstar * v2;
        Eabs += (real)0.5L * (real)mstar * v2;
        real l[3] = {xs[1] * vs[2] - xs[2] * vs[1], xs[2] * vs[0] - xs[0] * vs[2], xs[0] * vs[1] - xs[1] * vs[0]};
        for (int c = 0; c < 3; ++c) { L[c] += (real)mstar * l[c]; Labs[c] += R_FABS((real)mstar * l[c]); }
    }
    real Up = 0;
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : Up)
    for (int i = 0; i < nbig; ++i) {
        real acc = 0;
        for (int j = i + 1; j < nb; ++j) {
            real d2 = 0;
            for (int c = 0; c < 3; ++c) {
                real d = X_(x, c, i) - X_(x, c, j);
                d2 += d * d;
            }
            if (d2 > 0) acc += (real)mass[j] / R_SQRT(d2);
        }
        Up += (real)G * (real)mass[i] * acc;
    }
    Eabs += Up;
    Up = -Up;
    out[0] = (double)T; out[1] = (double)Us; out[2] = (double)Up; out[3] = (double)(T + Us + Up);
    for (int c = 0; c < 3; ++c) { out[4 + c] = (double)L[c]; out[8 + c] = (double)Labs[c]; }
    out[7] = (double)Eabs;
    return 0;
}

/* ---------------------------------------------------------------------------
 * Close-encounter resolution (the paper's mdt_hkce: "restore x and v to the
 * state before the call of arxes_drift using x0 and [v0] ... <integrate close encounters on CPU>";
 * PAPER.md:104 fn. 14: "switch to the slower Bulirsch-Stoer integration scheme to advance the
 * interaction and Keplerian Hamiltonians of the bodies involved in the close encounter").
 * The paper keeps this on the host and prints no algorithm; readings X-1..X-5:
 *   X-1 the bodies involved = every endpoint of the encounter pair list.  The connected components of
 *       the pair graph share no listed pair, so their equations of motion (X-2) are decoupled: each
 *       component is integrated as its own system, with its own step control, from the snapshot x0, v0
 *       over h (the parent code makes one mdt_hkce call for all of them; the solutions agree to the
 *       tolerance, and a tight pair no longer forces its small steps on a giant's hundred neighbours);
 *       all other bodies keep their Kepler-drift result
 *   X-2 equations of motion: dx/dt = v, dv/dt = -mu x/|x|^3 + sum over the LISTED pairs (i,j) that
 *       contain the body of gm_other (1 - K(r; rc)) (x_other - x_i)/r^3 - the complement of the
 *       K-weighted kick (A-1..A-5), so kick + encounter solve see the full Newtonian pair force
 *   X-3 integrator: Gragg's modified midpoint with n_k = 2, 4, .., 16 substeps, polynomial
 *       (Aitken-Neville) extrapolation in (H/n)^2; error of column k = max over components of
 *       |T_kk - T_k,k-1| / scale, scale = |x_i| (positions) and |v_i| (velocities) of that body at
 *       the start of the BS step; accepted when <= tol
 *   X-4 step control by column only: accepted at column k <= 3: H_next = 2 H; k <= 5: H; else H/2;
 *       no column accepted: H/2 and retry (40 halvings in a row are a failure: the bodies keep the
 *       drift result); H never exceeds what is left of h
 *   X-5 pairs summed in list order per body; coincident bodies contribute 0
 * ------------------------------------------------------------------------- */
#define BS_KMAX 8

typedef struct {
    int n;                 /* bodies in the system */
    int np;                /* pairs */
    const int *pi, *pj;    /* local body indices of each pair */
    const real *gm, *rc;   /* per local body */
    real mu;
} enc_sys;

/* f(y): y = [x(3n) | v(3n)] body-major (3 per body) */
static void enc_rhs(const enc_sys *s, const real *y, real *f)
{
    const int n = s->n;
    const real *X = y, *V = y + 3 * n;
    real *dX = f, *dV = f + 3 * n;
    for (int b = 0; b < n; ++b) {
        real r2 = X[3 * b] * X[3 * b] + X[3 * b + 1] * X[3 * b + 1] + X[3 * b + 2] * X[3 * b + 2];
        real r = R_SQRT(r2);
        real w = -s->mu / (r2 * r);
        for (int c = 0; c < 3; ++c) { dX[3 * b + c] = V[3 * b + c]; dV[3 * b + c] = w * X[3 * b + c]; }
    }
    for (int p = 0; p < s->np; ++p) {                       /* list order: fixed summation order per body */
        const int i = s->pi[p], j = s->pj[p];
        real d[3], s2 = 0;
        for (int c = 0; c < 3; ++c) { d[c] = X[3 * j + c] - X[3 * i + c]; s2 += d[c] * d[c]; }
        if (!(s2 > 0)) continue;
        real rc = rmax(s->rc[i], s->rc[j]);
        real K = changeover_s2(s2, rc);
        real u = ((real)1 - K) / (s2 * R_SQRT(s2));
        for (int c = 0; c < 3; ++c) {
            dV[3 * i + c] += s->gm[j] * u * d[c];
            dV[3 * j + c] -= s->gm[i] * u * d[c];
        }
    }
}

/* y over H with nsub modified-midpoint substeps -> out */
static void enc_midpoint(const enc_sys *s, const real *y, real H, int nsub, real *out, real *z0, real *z1, real *f)
{
    const int m = 6 * s->n;
    const real hs = H / (real)nsub;
    enc_rhs(s, y, f);
    for (int c = 0; c < m; ++c) { z0[c] = y[c]; z1[c] = y[c] + hs * f[c]; }
    for (int k = 1; k < nsub; ++k) {
        enc_rhs(s, z1, f);
        for (int c = 0; c < m; ++c) {
            real t = z0[c] + (real)2 * hs * f[c];
            z0[c] = z1[c]; z1[c] = t;
        }
    }
    enc_rhs(s, z1, f);
    for (int c = 0; c < m; ++c) out[c] = (real)0.5L * (z0[c] + z1[c] + hs * f[c]);
}

/* One system (X-1: one connected component of the pair graph): its bodies are the endpoints of `pairs`.
 * stats (nullable, 4 ints): bodies in the system, BS steps accepted, force evaluations, 1 if failed.
 * Returns 0, or 1 if the integration failed (x, v of its bodies untouched). */
static int resolve_system(int nb, int ld, double mu, const double *gm, const double *rcrit, double h,
                   const double *x0, const double *v0, double *x, double *v,
                   const int32_t *pairs, int64_t npairs, double tol, int32_t *stats)
{
    if (nb < 0 || ld < nb || npairs < 0 || !(tol > 0) || h == 0) return -1;
    if (stats) stats[0] = stats[1] = stats[2] = stats[3] = 0;
    if (npairs == 0) return 0;
    /* X-1: the system = sorted unique endpoints */
    int *loc = (int *)malloc(sizeof(int) * (size_t)nb);
    for (int b = 0; b < nb; ++b) loc[b] = -1;
    for (int64_t p = 0; p < npairs; ++p) { loc[pairs[2 * p]] = 0; loc[pairs[2 * p + 1]] = 0; }
    int n = 0;
    for (int b = 0; b < nb; ++b) if (loc[b] == 0) loc[b] = n++;
    int *body = (int *)malloc(sizeof(int) * (size_t)n);
    for (int b = 0; b < nb; ++b) if (loc[b] >= 0) body[loc[b]] = b;
    int *pi = (int *)malloc(sizeof(int) * (size_t)npairs), *pj = (int *)malloc(sizeof(int) * (size_t)npairs);
    for (int64_t p = 0; p < npairs; ++p) { pi[p] = loc[pairs[2 * p]]; pj[p] = loc[pairs[2 * p + 1]]; }
    const int m = 6 * n;
    real *g = (real *)malloc(sizeof(real) * (size_t)n), *rc = (real *)malloc(sizeof(real) * (size_t)n);
    real *y = (real *)malloc(sizeof(real) * (size_t)m * (BS_KMAX + 6));
    real *z0 = y + m, *z1 = z0 + m, *f = z1 + m, *scale = f + m, *res = scale + m, *T = res + m;  /* T: BS_KMAX rows */
    for (int k = 0; k < n; ++k) {
        g[k] = (real)gm[body[k]]; rc[k] = (real)rcrit[body[k]];
        for (int c = 0; c < 3; ++c) { y[3 * k + c] = X_(x0, c, body[k]); y[3 * n + 3 * k + c] = X_(v0, c, body[k]); }
    }
    enc_sys s = {n, (int)npairs, pi, pj, g, rc, (real)mu};
    const real hh = (real)h;
    real t = 0, H = hh;
    int fail = 0, nacc = 0, halvings = 0;
    long nrhs = 0;
    while (!fail) {
        const real rem = hh - t;
        if (R_FABS(rem) <= (real)4 * R_EPS * R_FABS(hh)) break;
        int last = 0;
        if (R_FABS(H) >= R_FABS(rem)) { H = rem; last = 1; }
        for (int k = 0; k < n; ++k) {                          /* X-3 scale: |x_i|, |v_i| at the start of the step */
            real sx = 0, sv = 0;
            for (int c = 0; c < 3; ++c) { sx += y[3 * k + c] * y[3 * k + c]; sv += y[3 * n + 3 * k + c] * y[3 * n + 3 * k + c]; }
            sx = R_SQRT(sx); sv = R_SQRT(sv);
            for (int c = 0; c < 3; ++c) { scale[3 * k + c] = sx; scale[3 * n + 3 * k + c] = sv; }
        }
        int acc_col = -1;
        for (int k = 0; k < BS_KMAX; ++k) {
            const int nsub = 2 * (k + 1);
            enc_midpoint(&s, y, H, nsub, res, z0, z1, f);
            nrhs += nsub + 1;
            /* Aitken-Neville per component: T[c][j] holds row k-1 (T_{k-1,j}) and is overwritten with row k */
            real err = 0;
            for (int c = 0; c < m; ++c) {
                real cur[BS_KMAX], *old = T + (size_t)c * BS_KMAX;   /* old[j] = T_{k-1, j} */
                cur[0] = res[c];
                for (int j = 1; j <= k; ++j) {
                    real ratio = (real)(2 * (k + 1)) / (real)(2 * (k - j + 1));
                    cur[j] = cur[j - 1] + (cur[j - 1] - old[j - 1]) / (ratio * ratio - (real)1);
                }
                if (k >= 1) {
                    real e = R_FABS(cur[k] - cur[k - 1]);
                    real sc = scale[c];
                    e = sc > 0 ? e / sc : (e > 0 ? (real)1e300 : (real)0);
                    if (e > err) err = e;
                }
                for (int j = 0; j <= k; ++j) old[j] = cur[j];
            }
            if (k >= 1 && err <= (real)tol) { acc_col = k; break; }
        }
        if (acc_col < 0) {                                     /* X-4: no column accepted */
            H *= (real)0.5L;
            if (++halvings > 40) fail = 1;
            continue;
        }
        for (int c = 0; c < m; ++c) y[c] = T[(size_t)c * BS_KMAX + acc_col];
        t = last ? hh : t + H;
        ++nacc;
        halvings = 0;                                          /* X-4: 40 CONSECUTIVE halvings are a failure */
        if (acc_col <= 3) H *= (real)2; else if (acc_col > 5) H *= (real)0.5L;
    }
    if (!fail) {
        for (int k = 0; k < n; ++k)
            for (int c = 0; c < 3; ++c) {
                x[(size_t)c * ld + body[k]] = (double)y[3 * k + c];
                v[(size_t)c * ld + body[k]] = (double)y[3 * n + 3 * k + c];
            }
    }
    if (stats) { stats[0] = n; stats[1] = nacc; stats[2] = (int32_t)nrhs; stats[3] = fail; }
    free(loc); free(body); free(pi); free(pj); free(g); free(rc); free(y);
    return fail;
}

/* pairs: npairs x 2 (i, j) body indices as mo_encounters lists them.  x, v: the drifted state, in/out.
 * X-1: union-find over the pairs; components taken in ascending order of their smallest body, each
 * with its pairs in list order.  stats (nullable, 4 ints): bodies in all systems, BS steps accepted
 * (summed over the components), force evaluations (summed), number of failed components.
 * Returns 0, or 1 if a component failed (its bodies keep the drift result). */
static int uf_find(int *par, int a) { while (par[a] != a) { par[a] = par[par[a]]; a = par[a]; } return a; }

int oracle_resolve(int nb, int ld, double mu, const double *gm, const double *rcrit, double h,
                   const double *x0, const double *v0, double *x, double *v,
                   const int32_t *pairs, int64_t npairs, double tol, int32_t *stats)
{
    if (nb < 0 || ld < nb || npairs < 0 || !(tol > 0) || h == 0) return -1;
    if (stats) stats[0] = stats[1] = stats[2] = stats[3] = 0;
    if (npairs == 0) return 0;
    int *par = (int *)malloc(sizeof(int) * (size_t)nb);
    for (int b = 0; b < nb; ++b) par[b] = b;
    for (int64_t p = 0; p < npairs; ++p) {
        int a = uf_find(par, pairs[2 * p]), b = uf_find(par, pairs[2 * p + 1]);
        if (a != b) { if (a < b) par[b] = a; else par[a] = b; }      /* root = smallest body of the component */
    }
    int32_t *sub = (int32_t *)malloc(sizeof(int32_t) * 2 * (size_t)npairs);
    char *done = (char *)calloc((size_t)npairs, 1);
    int anyfail = 0;
    for (int64_t p0 = 0; p0 < npairs; ++p0) {                        /* list sorted by (i, j): roots come up in ascending order */
        if (done[p0]) continue;
        const int root = uf_find(par, pairs[2 * p0]);
        int64_t ns = 0;
        for (int64_t p = p0; p < npairs; ++p)
            if (!done[p] && uf_find(par, pairs[2 * p]) == root) {
                sub[2 * ns] = pairs[2 * p]; sub[2 * ns + 1] = pairs[2 * p + 1]; ++ns; done[p] = 1;
            }
        int32_t st[4] = {0, 0, 0, 0};
        int f = resolve_system(nb, ld, mu, gm, rcrit, h, x0, v0, x, v, sub, ns, tol, st);
        if (stats) { stats[0] += st[0]; stats[1] += st[1]; stats[2] += st[2]; stats[3] += st[3]; }
        anyfail |= (f != 0);
    }
    free(par); free(sub); free(done);
    return anyfail;
}
