/*
 * rfoe_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU FP64 implementation of the recursive Fermi-operator
 * expansion (RFOE) hot path of arXiv 2301.04642, written from the paper.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use it.
 * It shares no code, header, table or helper with the CUDA library under
 * paper_2301_04642_b200/csrc/ and neither includes the other.
 *
 * What it follows (PAPER.md line : section):
 *   - X_{n+1} = X_n +/- (X_n - X_n^2), i.e. X^2 or 2X - X^2, sign chosen so that the trace
 *     of X_{n+1} lands nearer N_occ                                 PAPER.md:35-39 (sec. II.B.1, Eq. 1)
 *   - Tr(X) by diagonal traversal, Tr(X^2) = ||X||_F^2      PAPER.md:72    (sec. III.B)
 *   - RelTr = trace change relative to the previous iterate PAPER.md:64, 92 (sec. III.A, IV)
 *   - mixed precision: FP32 steps far from convergence,
 *     FP64 afterwards, switch tied to RelTr
 *   - truncated expansion G_m (T-RFOE): exactly m steps, no
 *     convergence test (variants ORC_TRUNC, ORC_TRUNC_MIXED) PAPER.md:47-52 (sec. II.B.3, Eq. 2)
 *   - accelerated (shifted/scaled) SP2 from HOMO/LUMO, in
 *     the unexpanded form "shift and scale, then SP2"       PAPER.md:43    (sec. II.B.2)
 *   - D = theta(mu I - H): a projector, eigenvalues 0/1     PAPER.md:27    (sec. II.A)
 * Where the paper is silent the readings R1..R16 of DESIGN.md are taken (initial affine map with
 * Gershgorin bounds, tie rule, stop rules A and B, the McWeeny-style switch).
 *
 * Arithmetic rules (so a reader can check it by eye): every product and sum is a separate
 * IEEE-754 double operation (compile with -ffp-contract=off, no -ffast-math); X_n^2 is the
 * naive triple loop with the contraction index l ascending.  rfoe_oracle_square_ijk is the literal
 * i-j-l loop nest; rfoe_oracle_square is the same arithmetic with the loops interchanged
 * (i-l-j, upper triangle, then mirrored) which is faster and bit-identical -- each Y_ij still adds
 * the products X_il*X_lj one at a time in ascending l; a CPU test pins the two to each other.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): Jacobi-eigendecomposition projector on tiny
 * inputs; construction-exact projector Q_occ Q_occ^T; diagonal-H closed form (scalar recursion);
 * per-step invariants; scalar eigenvalue-space model for branch strings and iteration counts;
 * the paper's printed iteration counts on the paper's matrix; the FP32 product
 * bit-for-bit against a numpy.float32 loop; the mixed schedule's phase switches and the out-of-range behaviour of
 * the sign rule on diagonal matrices worked by hand; T-RFOE against the exact Fermi-Dirac matrix.
 * Rayleigh-Ritz / apply / density (NEXT-4): pinned by an invariant-subspace construction against an
 * explicit eigendecomposition (numpy eigh and the Jacobi projector), sum rho = N_occ, and closed forms.
 * Not pinned: the exact bit patterns of X_n (the paper prints no worked example) -- "parity
 * unpinned" for bits, covered by tolerances.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_MAX_STEPS 256

enum { ORC_SP2 = 0, ORC_MCWEENY = 1, ORC_SP2_MIXED = 2, ORC_SP2_ACCEL = 3, ORC_TRUNC = 4, ORC_TRUNC_MIXED = 5 };
enum { ORC_RULE_A = 0, ORC_RULE_B = 1 };

typedef struct {
    /* inputs */
    int32_t variant;      /* ORC_* */
    int32_t stop_rule;    /* ORC_RULE_A: e_n = ||X_n^2 - X_n||_F <= tol ; ORC_RULE_B: RelTr <= tol */
    int32_t max_iter;     /* cap on recursion steps (<= ORACLE_MAX_STEPS) */
    int32_t use_bounds;   /* 1: take emin/emax below instead of Gershgorin */
    double tol;
    double emin, emax;    /* in: override when use_bounds; out: the bounds used */
    double mixed_head;    /* mixed: FP64 while (t - s) >= mixed_head  (0 => no FP64 head, paper schedule) */
    double mixed_reltr;   /* mixed: FP32 steps until RelTr <= mixed_reltr (paper: 5e-4), then FP64 */
    double homo, lumo;    /* accelerated SP2: eigenvalue estimates of H (lumo > homo) */
    /* outputs */
    int32_t iterations;   /* recursion steps taken */
    int32_t multiplications;
    int32_t mcweeny_steps;
    int32_t fp32_steps;
    int32_t converged;
    int32_t pad_;
    double tr_PH;         /* sum_ij P_ij H_ij */
    double t[ORACLE_MAX_STEPS + 1];   /* t[n] = Tr X_n */
    double s[ORACLE_MAX_STEPS + 1];   /* s[n] = sum_ij X_n,ij^2 */
    double e[ORACLE_MAX_STEPS];       /* e[n] = ||X_n^2 - X_n||_F */
    double reltr[ORACLE_MAX_STEPS];   /* |t[n+1]-t[n]| / |t[n]| */
    char branch[ORACLE_MAX_STEPS + 1];/* 'S' (X^2), 'L' (2X - X^2), 'M' (McWeeny), lower case = FP32 step */
} oracle_run_t;

/* ---- O1: Gershgorin bounds (reading R3) ------------------------------------------------- */
void rfoe_oracle_bounds(const double* H, int64_t k, double* emin, double* emax)
{
    double lo = 0.0, hi = 0.0;
    for (int64_t i = 0; i < k; ++i) {
        double r = 0.0;
        for (int64_t j = 0; j < k; ++j)
            if (j != i) r = r + fabs(H[i * k + j]);
        double a = H[i * k + i] - r, b = H[i * k + i] + r;
        if (i == 0 || a < lo) lo = a;
        if (i == 0 || b > hi) hi = b;
    }
    *emin = lo;
    *emax = hi;
}

/* ---- O2: affine initial map X0 = (emax I - H)/(emax - emin) (reading R2; true division) --- */
void rfoe_oracle_affine(const double* H, int64_t k, double emin, double emax, double* X)
{
    double w = emax - emin;
    for (int64_t i = 0; i < k; ++i)
        for (int64_t j = 0; j < k; ++j) {
            double num = (i == j) ? (emax - H[i * k + j]) : (-H[i * k + j]);
            X[i * k + j] = num / w;
        }
}

/* ---- O3: scalars.  Row sums first, then rows ascending (a fixed order) ------------------- */
double rfoe_oracle_trace(const double* X, int64_t k)
{
    double t = 0.0;
    for (int64_t i = 0; i < k; ++i) t = t + X[i * k + i];
    return t;
}

double rfoe_oracle_sumsq(const double* X, int64_t k)
{
    double s = 0.0;
    for (int64_t i = 0; i < k; ++i) {
        double r = 0.0;
        for (int64_t j = 0; j < k; ++j) r = r + X[i * k + j] * X[i * k + j];
        s = s + r;
    }
    return s;
}

static double sumsq_diff(const double* Y, const double* X, int64_t k)
{
    double s = 0.0;
    for (int64_t i = 0; i < k; ++i) {
        double r = 0.0;
        for (int64_t j = 0; j < k; ++j) {
            double d = Y[i * k + j] - X[i * k + j];
            r = r + d * d;
        }
        s = s + r;
    }
    return s;
}

/* ---- naive products ---------------------------------------------------------------------- */
/* literal: Y_ij = sum_{l=0..k-1} A_il * B_lj, l ascending */
void rfoe_oracle_matmul_ijk(const double* A, const double* B, int64_t k, double* Y)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < k; ++i)
        for (int64_t j = 0; j < k; ++j) {
            double acc = 0.0;
            for (int64_t l = 0; l < k; ++l) acc = acc + A[i * k + l] * B[l * k + j];
            Y[i * k + j] = acc;
        }
}

void rfoe_oracle_square_ijk(const double* X, int64_t k, double* Y)
{
    rfoe_oracle_matmul_ijk(X, X, k, Y);
}

/* same arithmetic, loops interchanged (i, l, j): row Y_i accumulates X_il * (row l of B), l ascending.
 * upper != 0: only j >= i is computed and the result mirrored (valid when the exact product is
 * symmetric AND A, B are bitwise symmetric and A == B, see header); else the full matrix. */
static void matmul_ilj(const double* A, const double* B, int64_t k, double* Y, int upper)
{
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t i = 0; i < k; ++i) {
        int64_t j0 = upper ? i : 0;
        double* y = Y + i * k;
        for (int64_t j = j0; j < k; ++j) y[j] = 0.0;
        for (int64_t l = 0; l < k; ++l) {
            const double a = A[i * k + l];
            const double* b = B + l * k;
            for (int64_t j = j0; j < k; ++j) y[j] = y[j] + a * b[j];
        }
    }
    if (upper) {
#pragma omp parallel for schedule(static)
        for (int64_t i = 1; i < k; ++i)
            for (int64_t j = 0; j < i; ++j) Y[i * k + j] = Y[j * k + i];
    }
}

void rfoe_oracle_square(const double* X, int64_t k, double* Y) { matmul_ilj(X, X, k, Y, 1); }
void rfoe_oracle_matmul(const double* A, const double* B, int64_t k, double* Y) { matmul_ilj(A, B, k, Y, 0); }

/* ---- tighter spectral bounds: m-step Lanczos estimate (reading R3b) ---------------------------------
 * The paper only says "spectral bound estimates"; Gershgorin (above) is the normative choice and
 * over-estimates the width of a dense rotated H^p ~50x at k=16384, which costs ~18 extra squarings.  This is the
 * standard alternative of Chebyshev-filtering codes: m steps of the Lanczos recursion from a fixed pseudo-random
 * start vector, T_m = tridiag(alpha, beta), and the bounds
 *        emin = theta_min(T_m) - beta_m,      emax = theta_max(T_m) + beta_m
 * (every Ritz value has an eigenvalue within beta_m; an estimator, safe in practice, not a proof -- the pins check
 * enclosure on the test matrices).  Plain recursion, no re-orthogonalisation, every sum in ascending index order:
 *   v_0 = s / ||s||,  s_i = hash(i) - 1/2   (32-bit integer hash below, the same on both sides of the parity test)
 *   w = H v_j;  alpha_j = v_j . w;  w -= alpha_j v_j + beta_j v_{j-1};  beta_{j+1} = ||w||;  v_{j+1} = w / beta_{j+1}
 * theta_min / theta_max by bisection on the Sturm count of T_m (200 halvings of a Gershgorin interval of T_m).
 * Returns the number of steps taken (< m if an invariant subspace was found: beta = 0, the bounds are then exact
 * for that subspace). alpha[m], beta[m+1] (beta[0] = 0) are written when not NULL. */
static double lanczos_start(uint32_t i)
{
    uint32_t x = i * 2654435761u + 0x9E3779B9u;
    x ^= x >> 16; x *= 0x85EBCA6Bu; x ^= x >> 13; x *= 0xC2B2AE35u; x ^= x >> 16;
    return (double)x * (1.0 / 4294967296.0) - 0.5;
}

static int sturm_count(const double* a, const double* b, int m, double x)   /* eigenvalues of T_m below x */
{
    int cnt = 0;
    double q = 1.0;
    for (int i = 0; i < m; ++i) {
        const double off = (i == 0) ? 0.0 : b[i] * b[i];
        q = a[i] - x - (i == 0 ? 0.0 : off / q);
        if (q == 0.0) q = 1e-300;
        if (q < 0.0) ++cnt;
    }
    return cnt;
}

int rfoe_oracle_bounds_lanczos(const double* H, int64_t k, int32_t m, double* emin, double* emax, double* alpha_out,
                               double* beta_out)
{
    if (m < 1) m = 1;
    if (m > 64) m = 64;
    if (m > k) m = (int32_t)k;
    double a[64] = {0.0}, b[65] = {0.0};
    double* v = (double*)malloc(sizeof(double) * (size_t)k);
    double* vp = (double*)malloc(sizeof(double) * (size_t)k);
    double* w = (double*)malloc(sizeof(double) * (size_t)k);
    double nrm2 = 0.0;
    for (int64_t i = 0; i < k; ++i) { v[i] = lanczos_start((uint32_t)i); vp[i] = 0.0; }
    for (int64_t i = 0; i < k; ++i) nrm2 = nrm2 + v[i] * v[i];
    const double n0 = sqrt(nrm2);
    for (int64_t i = 0; i < k; ++i) v[i] = v[i] / n0;
    b[0] = 0.0;
    int steps = 0;
    for (int j = 0; j < m; ++j) {
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < k; ++i) {
            double acc = 0.0;
            for (int64_t l = 0; l < k; ++l) acc = acc + H[i * k + l] * v[l];
            w[i] = acc;
        }
        double al = 0.0;
        for (int64_t i = 0; i < k; ++i) al = al + v[i] * w[i];
        a[j] = al;
        double s2 = 0.0;
        for (int64_t i = 0; i < k; ++i) {
            w[i] = (w[i] - al * v[i]) - b[j] * vp[i];
            s2 = s2 + w[i] * w[i];
        }
        b[j + 1] = sqrt(s2);
        steps = j + 1;
        if (!(b[j + 1] > 1e-14 * (fabs(al) + b[j]))) { b[j + 1] = 0.0; break; }
        for (int64_t i = 0; i < k; ++i) { vp[i] = v[i]; v[i] = w[i] / b[j + 1]; }
    }
    /* extreme eigenvalues of T_steps by bisection */
    double lo = a[0], hi = a[0];
    for (int i = 0; i < steps; ++i) {
        const double r = (i > 0 ? fabs(b[i]) : 0.0) + (i + 1 < steps ? fabs(b[i + 1]) : 0.0);
        if (a[i] - r < lo) lo = a[i] - r;
        if (a[i] + r > hi) hi = a[i] + r;
    }
    double l1 = lo, h1 = hi, l2 = lo, h2 = hi;
    for (int it = 0; it < 200; ++it) {
        const double m1 = 0.5 * (l1 + h1), m2 = 0.5 * (l2 + h2);
        if (sturm_count(a, b, steps, m1) >= 1) h1 = m1; else l1 = m1;          /* smallest eigenvalue */
        if (sturm_count(a, b, steps, m2) >= steps) h2 = m2; else l2 = m2;      /* largest eigenvalue */
    }
    *emin = 0.5 * (l1 + h1) - b[steps];
    *emax = 0.5 * (l2 + h2) + b[steps];
    if (alpha_out) for (int i = 0; i < steps; ++i) alpha_out[i] = a[i];
    if (beta_out) for (int i = 0; i <= steps; ++i) beta_out[i] = b[i];
    free(v); free(vp); free(w);
    return steps;
}

/* ---- steps either side of the expansion (reading R-RR) --------------
 * The paper's setting: "the discretized Kohn-Sham Hamiltonian matrix H of size M x M is
 * orthogonally projected onto a carefully constructed subspace ... (Rayleigh-Ritz step), and subsequently,
 * the resulting smaller dense projected Hamiltonian H^p of dimension k (<< M) is" handed to RFOE, which
 * "approximate[s] the density matrix in the subspace".  The paper prints neither step; they are written
 * here by their plain definitions for a basis stored one state per row (Psi: k x M, row pitch ld):
 *   project : H^p = Psi H Psi^T, given HPsi = (H Psi^T)^T (k x M, row j = H applied to state j):
 *             H^p_ij = sum_{m ascending} Psi_im * HPsi_jm for i <= j, then mirrored -- for symmetric H the
 *             exact H^p is symmetric, and rfoe_expand needs it bitwise symmetric, so the upper triangle is
 *             the definition (rfoe_oracle_project_full computes all k^2 sums for the pin that says so).
 *   apply   : Y = P Psi,  Y_im = sum_{j ascending} P_ij * Psi_jm      (the subspace density matrix applied
 *             to the basis; Psi^T Y is the density matrix in the full M-dimensional space)
 *   density : rho_m = sum_{i ascending} Psi_im * Y_im = (Psi^T P Psi)_mm (its diagonal: the electron
 *             density on the M degrees of freedom, per spin).  sum_m rho_m = Tr P = N_occ for orthonormal Psi. */
void rfoe_oracle_project_full(const double* Psi, const double* HPsi, int64_t k, int64_t M, int64_t ld, double* Hp)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < k; ++i)
        for (int64_t j = 0; j < k; ++j) {
            double acc = 0.0;
            for (int64_t m = 0; m < M; ++m) acc = acc + Psi[i * ld + m] * HPsi[j * ld + m];
            Hp[i * k + j] = acc;
        }
}

void rfoe_oracle_project(const double* Psi, const double* HPsi, int64_t k, int64_t M, int64_t ld, double* Hp)
{
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t i = 0; i < k; ++i)
        for (int64_t j = i; j < k; ++j) {
            double acc = 0.0;
            for (int64_t m = 0; m < M; ++m) acc = acc + Psi[i * ld + m] * HPsi[j * ld + m];
            Hp[i * k + j] = acc;
        }
    for (int64_t i = 1; i < k; ++i)
        for (int64_t j = 0; j < i; ++j) Hp[i * k + j] = Hp[j * k + i];
}

void rfoe_oracle_apply(const double* P, const double* Psi, int64_t k, int64_t M, int64_t ld, double* Y)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < k; ++i) {
        double* y = Y + i * ld;
        for (int64_t m = 0; m < M; ++m) y[m] = 0.0;
        for (int64_t j = 0; j < k; ++j) {          /* j ascending for every Y_im */
            const double p = P[i * k + j];
            const double* q = Psi + j * ld;
            for (int64_t m = 0; m < M; ++m) y[m] = y[m] + p * q[m];
        }
    }
}

void rfoe_oracle_density(const double* Psi, const double* Y, int64_t k, int64_t M, int64_t ld, double* rho)
{
    for (int64_t m = 0; m < M; ++m) rho[m] = 0.0;
    for (int64_t i = 0; i < k; ++i)                /* i ascending for every rho_m */
        for (int64_t m = 0; m < M; ++m) rho[m] = rho[m] + Psi[i * ld + m] * Y[i * ld + m];
}

/* ---- FP32 step of the mixed variants ("far away from RFOE convergence ... the floating point
 * operations can be performed in single precision (FP32)"): X rounded to float, every product and every sum a
 * separate IEEE binary32 operation, l ascending.  Pinned bit-for-bit against a numpy.float32 triple loop
 * (tests/test_oracle_pins.py::test_square_f32_bits).  xf, yf: caller-provided k*k float scratch. */
void rfoe_oracle_square_f32(const double* X, int64_t k, double* Y, float* xf, float* yf)
{
    for (int64_t i = 0; i < k * k; ++i) xf[i] = (float)X[i];
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t i = 0; i < k; ++i) {
        float* y = yf + i * k;
        for (int64_t j = i; j < k; ++j) y[j] = 0.0f;
        for (int64_t l = 0; l < k; ++l) {
            const float a = xf[i * k + l];
            const float* b = xf + l * k;
            for (int64_t j = i; j < k; ++j) y[j] = y[j] + a * b[j];
        }
    }
    for (int64_t i = 0; i < k; ++i)
        for (int64_t j = i; j < k; ++j) {
            Y[i * k + j] = (double)yf[i * k + j];
            Y[j * k + i] = (double)yf[i * k + j];
        }
}

int rfoe_oracle_is_symmetric(const double* X, int64_t k)
{
    for (int64_t i = 0; i < k; ++i)
        for (int64_t j = i + 1; j < k; ++j)
            if (memcmp(&X[i * k + j], &X[j * k + i], sizeof(double)) != 0) return 0;
    return 1;
}

/* ---- the sign of PAPER.md:39 ----------------------------------------------------------------------------
 * "The +/- sign is chosen to adjust the trace of X_{n+1} in each projection such that it converges to N_occ":
 * of the two candidate next iterates, take the one whose trace lands nearer N_occ; a tie takes the "+" sign
 * (2X - X^2; readings R4, R5).  For a spectrum inside [0,1] this is "X^2 iff Tr X_n > N_occ" (pinned by
 * test_step_invariants); when rounding has pushed an eigenvalue outside [0,1] it is the branch that maps it back
 * (pinned by test_sign_rule_repairs_out_of_range_eigenvalue).  Returns 1 for the squaring-type candidate. */
static int nearer_nocc(double trace_if_squared, double trace_if_other, double nocc)
{
    return fabs(trace_if_squared - nocc) < fabs(trace_if_other - nocc);
}

/* A-Z-RFOE: "shifting and scaling of the SP2 projection polynomials ... based on HOMO ... and LUMO
 * ... eigenvalues".  Reading R-ACC, written UNEXPANDED, i.e. as the paper's words say -- first shift
 * and scale, then apply the SP2 polynomial:
 *     squaring type:   Y = (1 - a) I + a X,  X' = Y^2,          a = 2 / (2 - lumo_img)
 *     other type:      Y = a X,              X' = 2 Y - Y^2,    a = 2 / (1 + homo_img)
 * lumo_img / homo_img are the images of the LUMO / HOMO eigenvalue under all maps applied so far. */
static void shift_scale(const double* X, int64_t k, double a, double shift, double* Y)
{
    for (int64_t i = 0; i < k; ++i)
        for (int64_t j = 0; j < k; ++j) {
            double v = a * X[i * k + j];
            Y[i * k + j] = (i == j) ? shift + v : v;
        }
}
static double poly_squaring(double x, double a) { double y = (1.0 - a) + a * x; return y * y; }
static double poly_other(double x, double a) { double y = a * x; return 2.0 * y - y * y; }

/* ---- O4/O5: the expansion ---------------------------------------------------------------- */
/* returns 0 on success (converged, truncated as asked, or max_iter reached; see run->converged),
 * -1 bad arguments, -2 H not bitwise symmetric, -3 empty bounds, -4 out of memory,
 * -5 accelerated variant: HOMO / LUMO estimates not inside the spectral bounds (emin <= homo < lumo <= emax) */
int rfoe_oracle_expand(const double* H, int64_t k, int64_t nocc, oracle_run_t* run, double* P)
{
    if (!H || !P || !run || k < 1 || nocc < 0 || nocc > k) return -1;
    if (run->max_iter < 0 || run->max_iter > ORACLE_MAX_STEPS) return -1;
    if (run->variant < ORC_SP2 || run->variant > ORC_TRUNC_MIXED) return -1;
    if (!rfoe_oracle_is_symmetric(H, k)) return -2;

    const int accel = (run->variant == ORC_SP2_ACCEL);
    const int mixed = (run->variant == ORC_SP2_MIXED || run->variant == ORC_TRUNC_MIXED);
    /* T-RFOE (Eq. 2): G_m = F_m(...F_0(H)...), "an intermediate function generated in Z-RFOE that
     * is obtained before the convergence": exactly max_iter = m steps, no convergence test */
    const int truncated = (run->variant == ORC_TRUNC || run->variant == ORC_TRUNC_MIXED);

    double emin, emax;
    if (run->use_bounds) { emin = run->emin; emax = run->emax; }
    else rfoe_oracle_bounds(H, k, &emin, &emax);
    run->emin = emin; run->emax = emax;
    if (!(emax > emin)) return -3;
    if (accel && !(emin <= run->homo && run->homo < run->lumo && run->lumo <= emax)) return -5;

    const size_t n2 = (size_t)k * (size_t)k;
    int rc = 0;
    double* X = (double*)malloc(n2 * sizeof(double));
    double* Y = (double*)malloc(n2 * sizeof(double));
    double* Z = (run->variant == ORC_MCWEENY || accel) ? (double*)malloc(n2 * sizeof(double)) : NULL;
    double* W = accel ? (double*)malloc(n2 * sizeof(double)) : NULL;
    float* xf = mixed ? (float*)malloc(n2 * sizeof(float)) : NULL;
    float* yf = mixed ? (float*)malloc(n2 * sizeof(float)) : NULL;
    if (!X || !Y || ((run->variant == ORC_MCWEENY || accel) && !Z) || (accel && !W) || (mixed && (!xf || !yf))) {
        rc = -4;
        goto cleanup;
    }

    rfoe_oracle_affine(H, k, emin, emax, X);
    double t = rfoe_oracle_trace(X, k), s = rfoe_oracle_sumsq(X, k);
    run->t[0] = t; run->s[0] = s;
    run->iterations = run->multiplications = run->mcweeny_steps = run->fp32_steps = 0;
    run->converged = 0;
    memset(run->branch, 0, sizeof(run->branch));

    double lumo_img = 0.0, homo_img = 1.0;     /* X0 = (emax I - H) / (emax - emin): occupied -> near 1 */
    if (accel) {
        lumo_img = (emax - run->lumo) / (emax - emin);
        homo_img = (emax - run->homo) / (emax - emin);
    }
    int mcweeny_phase = 0;
    int mixed_phase = mixed ? (run->mixed_head > 0.0 ? 0 : 1) : 2;  /* 0 FP64 head, 1 FP32, 2 FP64 */
    double reltr_prev = INFINITY;

    for (int n = 0; n < run->max_iter; ++n) {
        /* mixed schedule: FP32 steps "far away from RFOE convergence", "the number of initial FP32
         * iterations is linked to RelTr"; optional FP64 head while Tr X - Tr X^2 is still large (reading R-MIX) */
        if (mixed_phase == 0 && (t - s) < run->mixed_head) mixed_phase = 1;
        if (mixed_phase == 1 && reltr_prev <= run->mixed_reltr) mixed_phase = 2;
        const int fp32 = (mixed_phase == 1);
        if (run->variant == ORC_MCWEENY && !mcweeny_phase)
            if ((t - s) < 3.0 / 16.0 && fabs(t - (double)nocc) < 0.5) mcweeny_phase = 1;   /* R11 */

        /* Y = X_n^2 (every variant: e_n = ||X_n^2 - X_n||_F is measured on the step's input) */
        if (fp32) rfoe_oracle_square_f32(X, k, Y, xf, yf); else rfoe_oracle_square(X, k, Y);
        run->multiplications++;
        const double e = sqrt(sumsq_diff(Y, X, k));

        if (mcweeny_phase) {
            /* X' = 3 X^2 - 2 X^3, X^3 = (X^2) X as a second naive product */
            rfoe_oracle_matmul(Y, X, k, Z);
            run->multiplications++;
            for (int64_t i = 0; i < k; ++i)
                for (int64_t j = i; j < k; ++j) {
                    /* X^2 and X commute and are symmetric, but (X^2 X)_ij and (X^2 X)_ji need not round
                     * alike: keep the upper triangle and mirror it so that X stays bitwise symmetric */
                    double v = 3.0 * Y[i * k + j] - 2.0 * Z[i * k + j];
                    X[i * k + j] = v; X[j * k + i] = v;
                }
            run->branch[n] = 'M';
            run->mcweeny_steps++;
        } else if (accel) {
            /* both shifted-and-scaled candidates are formed (O(k^2)); their resulting traces follow from
             * Tr(A^2) = ||A||_F^2 for symmetric A; the chosen one is squared by the naive product.
             * (The product X_n^2 above only serves e_n here: the method needs one product per step and one is counted.) */
            const double aS = 2.0 / (2.0 - lumo_img), aO = 2.0 / (1.0 + homo_img);
            shift_scale(X, k, aS, 1.0 - aS, Z);                       /* Z = (1 - aS) I + aS X */
            shift_scale(X, k, aO, 0.0, W);                            /* W = aO X              */
            const double trace_if_squared = rfoe_oracle_sumsq(Z, k);                             /* Tr Z^2       */
            const double trace_if_other = 2.0 * rfoe_oracle_trace(W, k) - rfoe_oracle_sumsq(W, k); /* Tr(2W - W^2) */
            if (nearer_nocc(trace_if_squared, trace_if_other, (double)nocc)) {
                rfoe_oracle_square(Z, k, X);
                lumo_img = poly_squaring(lumo_img, aS);
                homo_img = poly_squaring(homo_img, aS);
                run->branch[n] = 'S';
            } else {
                rfoe_oracle_square(W, k, Y);
                for (size_t q = 0; q < n2; ++q) X[q] = 2.0 * W[q] - Y[q];
                lumo_img = poly_other(lumo_img, aO);
                homo_img = poly_other(homo_img, aO);
                run->branch[n] = 'L';
            }
        } else if (nearer_nocc(s, 2.0 * t - s, (double)nocc)) {       /* Tr X^2 = s, Tr(2X - X^2) = 2t - s */
            memcpy(X, Y, n2 * sizeof(double));
            run->branch[n] = fp32 ? 's' : 'S';
        } else {
            for (size_t q = 0; q < n2; ++q) X[q] = 2.0 * X[q] - Y[q];
            run->branch[n] = fp32 ? 'l' : 'L';
        }
        if (fp32) run->fp32_steps++;

        double t1 = rfoe_oracle_trace(X, k), s1 = rfoe_oracle_sumsq(X, k);
        double reltr = fabs(t1 - t) / fabs(t);
        run->e[n] = e; run->reltr[n] = reltr;
        run->t[n + 1] = t1; run->s[n + 1] = s1;
        t = t1; s = s1; reltr_prev = reltr;
        run->iterations = n + 1;
        /* mixed: an FP32 step never terminates the expansion (its e, RelTr sit on the FP32 floor) */
        if (!fp32 && !truncated) {
            if (run->stop_rule == ORC_RULE_A ? (e <= run->tol) : (reltr <= run->tol)) { run->converged = 1; break; }
        }
    }
    if (truncated) run->converged = (run->iterations == run->max_iter);   /* G_m delivered as asked */

    memcpy(P, X, n2 * sizeof(double));
    {
        double acc = 0.0;
        for (int64_t i = 0; i < k; ++i) {
            double r = 0.0;
            for (int64_t j = 0; j < k; ++j) r = r + P[i * k + j] * H[i * k + j];
            acc = acc + r;
        }
        run->tr_PH = acc;
    }
cleanup:
    free(X); free(Y); free(Z); free(W); free(xf); free(yf);
    return rc;
}

int rfoe_oracle_sizeof_run(void) { return (int)sizeof(oracle_run_t); }
int rfoe_oracle_max_steps(void) { return ORACLE_MAX_STEPS; }
