// Device-side control of the recursion (rows A3 + A6 of DESIGN.md): one 256-thread block sums the
// per-row / per-tile partials in a fixed order, appends the step to the history, applies the stop
// rule, chooses the next step's branch from Tr X_n vs N_occ and writes (i) the
// epilogue coefficients the next squaring reads from device memory and (ii) ONE word for the host
// (what to launch next) into mapped pinned memory -- the only host<->device traffic per step.
#pragma once
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include "sym_square.cuh"

namespace rfoe {

constexpr int CTRL_MAX_STEPS = 256;

enum Action : int { ACT_STOP = 0, ACT_SP2 = 1, ACT_MCWEENY = 2, ACT_SP2_FP32 = 3 };
enum Variant : int { VAR_SP2 = 0, VAR_MCWEENY = 1, VAR_MIXED = 2, VAR_ACCEL = 3, VAR_TRUNC = 4, VAR_TRUNC_MIXED = 5 };

struct Ctrl {
    // configuration (host -> device once per expansion)
    int variant, stop_rule, max_iter, kvalid;
    double nocc, tol;
    double mixed_head, mixed_reltr;
    double homo, lumo;
    // state
    int step;            // recursion steps completed
    int action;          // next action (mirrors the host word)
    int mcweeny_phase, mixed_phase;
    int multiplications, mcweeny_steps, fp32_steps, converged;
    int error, pad_;     // set by the first decision: 0 ok, 1 spectral bounds empty / not finite, 2 HOMO / LUMO estimates outside them
    double t, s, reltr_prev;
    double beta, bbar;   // accelerated SP2: images of LUMO / HOMO under the maps applied so far
    double emin, emax;
    double tr_PH;
    StepCoef coef;       // epilogue coefficients of the NEXT squaring: Out = c2 C + c1 E + c0 I
    StepCoef coef_aux;   // McWeeny: coefficients of the second product (3 Y - 2 Y X)
    // history
    double ht[CTRL_MAX_STEPS + 1], hs[CTRL_MAX_STEPS + 1], he[CTRL_MAX_STEPS], hreltr[CTRL_MAX_STEPS];
    char branch[CTRL_MAX_STEPS + 8];
};

// fixed-order block sum of n values read with a stride (in doubles); result valid in every thread
__device__ inline double block_sum_strided(const double* __restrict__ p, int n, int stride, double* sh)
{
    double v = 0.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) v += p[(size_t)i * stride];
    sh[threadIdx.x] = v;
    __syncthreads();
    for (int m = blockDim.x >> 1; m >= 1; m >>= 1) {
        if ((int)threadIdx.x < m) sh[threadIdx.x] += sh[threadIdx.x + m];
        __syncthreads();
    }
    const double r = sh[0];
    __syncthreads();
    return r;
}

// min / max of the Gershgorin discs -> bounds[0..1]  (A1, second pass)
__global__ void __launch_bounds__(256)
bounds_reduce_kernel(const double* __restrict__ row_lo, const double* __restrict__ row_hi, int k, double* __restrict__ bounds)
{
    __shared__ double slo[256], shi[256];
    double lo = INFINITY, hi = -INFINITY;
    int bad = 0;                       // fmin / fmax drop NaNs: a non-finite H^p must not yield finite bounds
    for (int i = threadIdx.x; i < k; i += 256) {
        const double a = row_lo[i], b = row_hi[i];
        bad |= (a != a) | (b != b);
        lo = fmin(lo, a);
        hi = fmax(hi, b);
    }
    bad = __syncthreads_or(bad);
    slo[threadIdx.x] = lo;
    shi[threadIdx.x] = hi;
    __syncthreads();
    for (int m = 128; m >= 1; m >>= 1) {
        if ((int)threadIdx.x < m) {
            slo[threadIdx.x] = fmin(slo[threadIdx.x], slo[threadIdx.x + m]);
            shi[threadIdx.x] = fmax(shi[threadIdx.x], shi[threadIdx.x + m]);
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        bounds[0] = bad ? NAN : slo[0];
        bounds[1] = bad ? NAN : shi[0];
    }
}

// choose the next action + coefficients from the current (t, s); thread 0 only
__device__ inline void decide_next(Ctrl* c)
{
    const double t = c->t, s = c->s;
    // "The +/- sign is chosen to adjust the trace of X_{n+1} ... such that it converges to N_occ":
    // the branch whose RESULTING trace is nearer N_occ, tie -> L (R4, R5).  Both candidate traces follow from
    // t = Tr X_n and s = Tr X_n^2 before the product.  Inside [0,1] this is "S iff t > N_occ"; it differs only
    // when rounding noise has pushed eigenvalues outside [0,1], where it picks the branch that maps them back.
    double trS = s, trL = 2.0 * t - s;
    if (c->variant == VAR_ACCEL) {
        const double aS = 2.0 / (2.0 - c->beta), aL = 2.0 / (1.0 + c->bbar);
        trS = aS * aS * s + 2.0 * aS * (1.0 - aS) * t + (1.0 - aS) * (1.0 - aS) * (double)c->kvalid;
        trL = 2.0 * aL * t - aL * aL * s;
    }
    const bool sq = fabs(trS - c->nocc) < fabs(trL - c->nocc);
    int action = ACT_SP2;
    if (c->variant == VAR_MCWEENY) {
        if (!c->mcweeny_phase && (t - s) < 3.0 / 16.0 && fabs(t - c->nocc) < 0.5) c->mcweeny_phase = 1;   // R11
        if (c->mcweeny_phase) action = ACT_MCWEENY;
    } else if (c->variant == VAR_MIXED || c->variant == VAR_TRUNC_MIXED) {
        if (c->mixed_phase == 0 && (t - s) < c->mixed_head) c->mixed_phase = 1;
        if (c->mixed_phase == 1 && c->reltr_prev <= c->mixed_reltr) c->mixed_phase = 2;
        if (c->mixed_phase == 1) action = ACT_SP2_FP32;
    }
    const int n = c->step;
    if (action == ACT_MCWEENY) {
        c->coef = StepCoef{1.0, 0.0, 0.0};              // Y = X^2
        c->coef_aux = StepCoef{-2.0, 3.0, 0.0};         // X' = 3 Y - 2 (Y X)
        c->branch[n] = 'M';
    } else if (c->variant == VAR_ACCEL) {
        if (sq) {
            const double a = 2.0 / (2.0 - c->beta);
            c->coef = StepCoef{a * a, 2.0 * a * (1.0 - a), (1.0 - a) * (1.0 - a)};
            double u = (1.0 - a) + a * c->beta;
            c->beta = u * u;
            u = (1.0 - a) + a * c->bbar;
            c->bbar = u * u;
        } else {
            const double a = 2.0 / (1.0 + c->bbar);
            c->coef = StepCoef{-(a * a), 2.0 * a, 0.0};
            c->beta = 2.0 * a * c->beta - a * a * c->beta * c->beta;
            c->bbar = 2.0 * a * c->bbar - a * a * c->bbar * c->bbar;
        }
        c->branch[n] = sq ? 'S' : 'L';
    } else {
        c->coef = sq ? StepCoef{1.0, 0.0, 0.0} : StepCoef{-1.0, 2.0, 0.0};
        c->branch[n] = (action == ACT_SP2_FP32) ? (sq ? 's' : 'l') : (sq ? 'S' : 'L');
    }
    c->action = action;
}

// first decision (thread 0): t_0, s_0 and the spectral bounds are known; validity of the bounds and (A-Z-RFOE) the
// images of LUMO / HOMO under the affine map are settled here, on the device, so that a launch sequence enqueued
// without a host round trip stops by itself on bad input
__device__ inline void control_begin(Ctrl* c, double t0, double s0, const double* __restrict__ bounds)
{
    const double emin = bounds[0], emax = bounds[1];
    c->emin = emin; c->emax = emax;
    c->t = t0; c->s = s0;
    c->ht[0] = t0; c->hs[0] = s0;
    c->step = 0;
    int err = 0;
    if (!(isfinite(emin) && isfinite(emax) && emax > emin)) err = 1;
    else if (c->variant == VAR_ACCEL) {
        if (!(emin <= c->homo && c->homo < c->lumo && c->lumo <= emax)) err = 2;
        c->beta = (emax - c->lumo) / (emax - emin);
        c->bbar = (emax - c->homo) / (emax - emin);
    }
    c->error = err;
    if (err || c->max_iter <= 0) c->action = ACT_STOP; else decide_next(c);
}

// one finished recursion step (thread 0): t_{n+1}, s_{n+1} and e_n^2 are the fixed-order sums of the step's records
__device__ inline void control_update(Ctrl* c, double t1, double s1, double e2)
{
    const int n = c->step;
    const int was_fp32 = (c->action == ACT_SP2_FP32);
    const double e = sqrt(e2);
    const double reltr = fabs(t1 - c->t) / fabs(c->t);
    c->he[n] = e; c->hreltr[n] = reltr;
    c->ht[n + 1] = t1; c->hs[n + 1] = s1;
    c->multiplications += (c->action == ACT_MCWEENY) ? 2 : 1;
    c->mcweeny_steps += (c->action == ACT_MCWEENY);
    c->fp32_steps += was_fp32;
    c->t = t1; c->s = s1; c->reltr_prev = reltr;
    c->step = n + 1;
    bool stop = false;
    const bool truncated = (c->variant == VAR_TRUNC || c->variant == VAR_TRUNC_MIXED);
    if (truncated) {   // T-RFOE: exactly max_iter = m steps, no convergence test; G_m delivered = success
        if (c->step >= c->max_iter) { stop = true; c->converged = 1; }
    } else if (!was_fp32) {   // an FP32 step never terminates the expansion (its e, RelTr sit on the FP32 floor)
        if (c->stop_rule == 0 ? (e <= c->tol) : (reltr <= c->tol)) { stop = true; c->converged = 1; }
    }
    if (!stop && c->step >= c->max_iter) stop = true;
    if (stop) c->action = ACT_STOP; else decide_next(c);
}

// mode 0: after the affine map (row_tr / row_ss hold k per-row values; bounds = the two device scalars) -> t_0, s_0,
//         first decision.
// mode 1: after a recursion step.  part_ts: tile records of the launch that wrote X_{n+1} (Tr, ||.||_F^2),
//         part_e: tile records of the squaring X_n^2 (||X_n^2 - X_n||_F^2); n_rec records each.
__global__ void __launch_bounds__(256)
control_kernel(Ctrl* __restrict__ c, int mode, const double* __restrict__ part_ts, const double* __restrict__ part_e,
               int n_rec, volatile int* __restrict__ host_word, const double* __restrict__ bounds)
{
    __shared__ double sh[256];
    if (mode == 0) {
        const double t0 = block_sum_strided(part_ts, n_rec, 1, sh);
        const double s0 = block_sum_strided(part_e, n_rec, 1, sh);
        if (threadIdx.x == 0) {
            control_begin(c, t0, s0, bounds);
            *host_word = c->action;
            __threadfence_system();
        }
        return;
    }
    const double t1 = block_sum_strided(part_ts + 0, n_rec, SQ_NPART, sh);
    const double s1 = block_sum_strided(part_ts + 1, n_rec, SQ_NPART, sh);
    const double e2 = block_sum_strided(part_e + 2, n_rec, SQ_NPART, sh);
    if (threadIdx.x == 0) {
        control_update(c, t1, s1, e2);
        *host_word = c->action;
        __threadfence_system();
    }
}

// tr(P H) from per-row values; also used for generic "sum k values" jobs (dst[0] = sum)
__global__ void __launch_bounds__(256)
sum_rows_kernel(const double* __restrict__ rows, int n, double* __restrict__ dst)
{
    __shared__ double sh[256];
    const double v = block_sum_strided(rows, n, 1, sh);
    if (threadIdx.x == 0) *dst = v;
}

// Tr X of a pitched work matrix (rfoe_square_reduced needs it for the shift)
__global__ void __launch_bounds__(256)
diag_sum_kernel(const double* __restrict__ X, int k, int ld, double* __restrict__ dst)
{
    __shared__ double sh[256];
    const double v = block_sum_strided(X, k, ld + 1, sh);
    if (threadIdx.x == 0) *dst = v;
}

// 5 scalars of one squaring launch (rfoe_square / rfoe_symm_product)
__global__ void __launch_bounds__(256)
sum_partials_kernel(const double* __restrict__ part, int n_rec, double* __restrict__ dst5)
{
    __shared__ double sh[256];
    for (int q = 0; q < 5; ++q) {
        const double v = block_sum_strided(part + q, n_rec, SQ_NPART, sh);
        if (threadIdx.x == 0) dst5[q] = v;
    }
}

}  // namespace rfoe
