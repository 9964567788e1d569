/*
 * rfoe.h -- C ABI of librfoe: recursive Fermi-operator expansion (RFOE) on one B200 (sm_100a).
 *
 * Problem statement (arXiv 2301.04642; sec. II.A, sec. III.A): given the dense
 * symmetric FP64 projected Kohn-Sham Hamiltonian H^p (k x k) and the number of occupied states
 * N_occ, produce the density matrix D = theta(mu I - H^p), i.e. the projector P onto the N_occ lowest
 * eigenvectors, WITHOUT diagonalising: a trace-steered recursion of dense matrix squarings
 * X_{n+1} = X_n^2 or 2 X_n - X_n^2 (SP2, Eq. 1) and the variants listed below.
 *
 * Conventions for every entry point
 *   - Matrices are contiguous row-major k x k FP64 with leading dimension k.  "device" pointers are
 *     CUDA device pointers owned by the caller (e.g. torch data_ptr()); "host" pointers are ordinary
 *     host memory.  The library never frees or keeps caller pointers after a call returns.
 *   - `stream` is a cudaStream_t (0 = the legacy default stream).  All device work of a call is
 *     issued on it.  Calls block the host until their result is complete (rfoe_expand reads one
 *     scalar per recursion step from the device).
 *   - Every function returns an rfoe_status_t.  There are no exceptions, no output on stdout/stderr
 *     and no CPU fallback: without a usable CUDA device rfoe_create fails with RFOE_ERR_CUDA.
 *   - A handle may be used by one host thread at a time.
 */
#ifndef RFOE_H_
#define RFOE_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rfoe_handle_s* rfoe_handle_t;
typedef struct CUstream_st* rfoe_stream_t; /* == cudaStream_t */

typedef enum {
    RFOE_OK = 0,
    RFOE_ERR_INVALID_ARG = 1,   /* null pointer, k < 1 or k > k_max, nocc outside (0,k), tol not finite/negative */
    RFOE_ERR_ALLOC = 2,         /* device or pinned allocation failed */
    RFOE_ERR_CUDA = 3,          /* a CUDA call failed; the cudaError_t is in rfoe_stats_t.cuda_error */
    RFOE_ERR_BAD_BOUNDS = 4,    /* eps_max <= eps_min (e.g. H^p is a multiple of the identity) or not finite */
    RFOE_ERR_NOT_SYMMETRIC = 5, /* H^p is not bitwise symmetric (the squaring X X^T relies on it) */
    RFOE_ERR_UNSUPPORTED = 6,   /* unknown variant / option, or device is not compute capability 10.x */
    RFOE_ERR_NOT_CONVERGED = 7, /* max_iter steps taken; P holds the last iterate, stats are complete */
    RFOE_ERR_NO_PEER_ACCESS = 8, /* sharded P2P setup: a peer's buffers cannot be mapped (cudaDeviceCanAccessPeer is false, or
                                   cudaIpcOpenMemHandle failed: cuda_error has the reason); use rfoe_expand_sharded instead */
    RFOE_ERR_STATIC_LIMIT = 9   /* rfoe_bounds_static: k > RFOE_STATIC_MAX_K, the size its fixed scratch array was built for */
} rfoe_status_t;

/* Recursion variants.
 *  SP2        Z-RFOE with second-order projection polynomials           PAPER.md:35-39 (sec. II.B.1)
 *  MCWEENY    SP2 until (Tr X - Tr X^2) < 3/16 and |Tr X - N_occ| < 1/2, then X <- 3X^2 - 2X^3
 *             (purification, cited only: PAPER.md:23; reading R11 in DESIGN.md)
 *  SP2_MIXED  reduced-precision (three FP16-part products on tcgen05, FP32 accumulate) squarings far from convergence, FP64 afterwards,
 *             switch tied to RelTr; optional FP64 head (RFOE_OPT_MIXED_HEAD)
 *  SP2_ACCEL  A-Z-RFOE: shifted-and-scaled SP2 polynomials from HOMO/LUMO estimates
 *                                                                       PAPER.md:43 (sec. II.B.2)
 *  TRUNC      T-RFOE, the paper's finite-temperature scheme: the truncated expansion        PAPER.md:47-52 (sec. II.B.3, Eq. 2)
 *             G_m(H^p) = F_m(...F_0(H^p)...), "an intermediate function generated in Z-RFOE that is obtained before the
 *             convergence", a smeared stand-in for the Fermi-Dirac matrix [exp(beta (H - mu I)) + I]^-1.
 *             Exactly m = RFOE_OPT_TRUNC_STEPS SP2 steps (default 30, the paper's "around 30" at 500 K), no
 *             convergence test, `tol` ignored; returns RFOE_OK with iterations == m and stats.trunc_steps == m.  The paper
 *             gives no m(beta) relation; DESIGN.md (reading R-TRUNC) tabulates the one measured on its matrix.
 *  TRUNC_MIXED  mixed-precision T-RFOE: the same m steps, reduced-precision ones until
 *             RelTr <= RFOE_OPT_MIXED_RELTR (and after the optional FP64 head), FP64 afterwards.
 * (SP2 with RFOE_OPT_MAX_ITER = m and tol = 0 runs the same m steps but reports RFOE_ERR_NOT_CONVERGED: that route is
 * a convergence failure by definition; TRUNC is the method of PAPER.md:47-52.) */
enum { RFOE_VARIANT_SP2 = 0, RFOE_VARIANT_MCWEENY = 1, RFOE_VARIANT_SP2_MIXED = 2, RFOE_VARIANT_SP2_ACCEL = 3,
       RFOE_VARIANT_TRUNC = 4, RFOE_VARIANT_TRUNC_MIXED = 5 };

/* Options (rfoe_set_option).  Values are doubles; integer options are rounded. */
enum {
    RFOE_OPT_STOP_RULE = 0,    /* 0 (default) rule A: stop after the step whose e_n = ||X_n^2 - X_n||_F <= tol;
                                  1 rule B (paper): RelTr_n = |Tr X_{n+1} - Tr X_n| / |Tr X_n| <= tol */
    RFOE_OPT_MAX_ITER = 1,     /* cap on recursion steps, 1..RFOE_MAX_STEPS (default 100) */
    RFOE_OPT_EPS_MIN = 2,      /* caller-supplied spectral bounds; used instead of Gershgorin when   */
    RFOE_OPT_EPS_MAX = 3,      /*   both are set and eps_max > eps_min.  NaN (default) = unset          */
    RFOE_OPT_CHECK_SYMMETRY = 4, /* 1 (default): one pass over H^p comparing (i,j) with (j,i) bitwise */
    RFOE_OPT_MIXED_HEAD = 5,   /* SP2_MIXED: FP64 while (Tr X - Tr X^2) >= value; 0 (default) = paper schedule */
    RFOE_OPT_MIXED_RELTR = 6,  /* SP2_MIXED: FP32 steps until RelTr <= value (default 5e-4) */
    RFOE_OPT_HOMO = 7,         /* SP2_ACCEL: estimate of the highest occupied eigenvalue of H^p */
    RFOE_OPT_LUMO = 8,         /* SP2_ACCEL: estimate of the lowest unoccupied eigenvalue of H^p */
    RFOE_OPT_LANCZOS_STEPS = 9, /* 0 (default): Gershgorin bounds in rfoe_expand; m in 1..64: rfoe_bounds_lanczos with m steps */
    RFOE_OPT_TRUNC_STEPS = 10, /* TRUNC / TRUNC_MIXED: the number m of recursion steps, 1..RFOE_MAX_STEPS (default 30) */
    RFOE_OPT_RESIDENT = 11,    /* 1 (default): expansions small enough to stay on chip (see rfoe_expand) run the WHOLE recursion
                                  in one persistent launch, no host round trip per step; 0: one launch sequence per step;
                                  2: as 1, but tiles cut between SMs are always finished in bands after a grid barrier (the
                                  form 1 picks outside k = 1792 ... 2816), never by their first holder (tests, A/B) */
    RFOE_OPT_REDUCED_PAIR = 12 /* 1 (default): reduced-precision products as CTA-pair MMAs (tcgen05.mma.cta_group::2, the shared
                                  row panel split between the two SMs of a TPC); 0: one CTA per tile with TMA multicast.
                                  The same products in the same order; results agree to the last bits of the FP32 sums */
};

#define RFOE_MAX_STEPS 256

typedef struct {
    int32_t status;          /* rfoe_status_t of the last rfoe_expand / rfoe_bounds */
    int32_t cuda_error;      /* last cudaError_t seen (0 = cudaSuccess) */
    int32_t variant;
    int32_t stop_rule;
    int32_t iterations;      /* recursion steps taken (= squarings of X_n) */
    int32_t multiplications; /* dense products launched (McWeeny steps take two) */
    int32_t mcweeny_steps;
    int32_t fp32_steps;
    int32_t converged;
    int32_t square_launches; /* launches of the symmetric squaring / product kernel */
    int32_t trunc_steps;     /* TRUNC / TRUNC_MIXED: the m asked for (0 for the other variants): iterations == trunc_steps
                                means "truncated on purpose", as opposed to status NOT_CONVERGED */
    int32_t resident;        /* 1 when the recursion ran as one persistent launch (RFOE_OPT_RESIDENT) */
    int64_t k;
    int64_t nocc;
    int64_t gpu_launches;    /* kernels launched by the last call */
    double tol;
    double eps_min, eps_max; /* the bounds used for X_0 */
    double tr_PH;            /* sum_ij P_ij H^p_ij (band energy) */
    double device_ms;        /* CUDA-event time of the last rfoe_expand on its stream */
    double square_ms;        /* CUDA-event time summed over its squaring / product kernel launches (persistent launch: the
                                steps as timed by CTA 0 with %globaltimer) */
    double resident_phase_ms[5]; /* persistent launch only, CTA 0's share of the steps: products, first grid barrier (the wait
                                for the slowest SM included), finishing of split tiles, second barrier, reductions + decision */
    double t[RFOE_MAX_STEPS + 1];   /* t[n] = Tr X_n */
    double s[RFOE_MAX_STEPS + 1];   /* s[n] = ||X_n||_F^2 = Tr X_n^2 */
    double e[RFOE_MAX_STEPS];       /* e[n] = ||X_n^2 - X_n||_F (idempotency error of the step's input) */
    double reltr[RFOE_MAX_STEPS];   /* |t[n+1] - t[n]| / |t[n]| */
    char branch[RFOE_MAX_STEPS + 8];/* per step: 'S' X^2, 'L' 2X - X^2, 'M' McWeeny; lower case = FP32 step */
} rfoe_stats_t;

/* Create a handle on CUDA device `device` able to expand matrices up to k_max x k_max.
 * Allocates (device) three zero-padded work matrices of ceil(k_max/128)*128 squared doubles (the third
 * lazily, on the first McWeeny call; two FP16 part matrices lazily on the first mixed call; further scratch lazily by
 * the projection / apply / sharded / Lanczos entry points), per-tile reduction scratch and one pinned host page.
 * Errors: INVALID_ARG (h null, k_max < 1), CUDA (no device / wrong device), UNSUPPORTED (not sm_100),
 * ALLOC. */
int rfoe_create(rfoe_handle_t* h, int device, int64_t k_max);

/* Gershgorin spectral bounds of H^p (reading R3; the paper only says "spectral bound estimates",
 * PAPER.md:56): eps_min = min_i (H_ii - r_i), eps_max = max_i (H_ii + r_i), r_i = sum_{j != i} |H_ij|.
 * Hp: device, k x k, read only.  eps_min / eps_max: HOST doubles, written on success.  Pure query. */
int rfoe_bounds(rfoe_handle_t h, const double* Hp, int64_t k, double* eps_min, double* eps_max, rfoe_stream_t stream);

/* The same Gershgorin bounds (row A1; reading R3) for callers that cannot allocate: code under CUDA graph
 * capture, serving loops and harnesses that forbid cudaMalloc.  No handle, no allocation: this call and everything
 * under it calls no cudaMalloc / cudaFree / allocating library routine.  The per-row disc ends (2 k doubles), which
 * rfoe_bounds keeps in handle memory, live in ONE file-scope `static __device__` array of 2 * RFOE_STATIC_MAX_K
 * doubles (512 KiB) that every GPU which loads the library holds until the process exits.
 *   Hp      device, k x k, read only, on the CURRENT device (cudaGetDevice); k <= RFOE_STATIC_MAX_K, else
 *           RFOE_ERR_STATIC_LIMIT and nothing is launched.
 *   bounds  DEVICE, 2 doubles, caller-owned: bounds[0] = eps_min, bounds[1] = eps_max (as rfoe_bounds: both NaN when H^p
 *           holds a NaN, -inf / +inf when it holds an infinity -- never finite for a non-finite H^p).
 *   cuda_error  host, may be null: the cudaError_t behind an RFOE_ERR_CUDA return.
 * Unlike the handle calls this one is ASYNCHRONOUS: it enqueues two kernels on `stream` and returns; `bounds` is valid
 * once the stream has passed them.  The first call on each device resolves the array's device address
 * (cudaGetSymbolAddress, which may load the module): make that call outside stream capture.
 * Every call on a device shares the one array, which keeps the last call's contents.  Nothing in it must start at
 * zero: a call writes entries [0, k) of both halves before it reads exactly those.  Calls that OVERLAP on the same GPU
 * (two streams, or two host threads) race on the array and give wrong bounds: serialise them (one stream, or events).
 * Results are bit for bit those of rfoe_bounds.
 * Errors: INVALID_ARG (null pointer, k < 1), STATIC_LIMIT, UNSUPPORTED (current device is not compute capability
 * 10.x), CUDA. */
#define RFOE_STATIC_MAX_K 32768
int rfoe_bounds_static(const double* Hp, int64_t k, double* bounds, rfoe_stream_t stream, int* cuda_error);

/* Tighter "spectral bound estimates" than Gershgorin's: m steps (1..64; 24 is plenty) of the Lanczos
 * recursion from a fixed pseudo-random start vector, T_m = tridiag(alpha, beta), and
 *     eps_min = theta_min(T_m) - beta_m,   eps_max = theta_max(T_m) + beta_m
 * (the estimator of Chebyshev-filtering codes: safe in practice, not a proof; reading R3b).  On a dense
 * rotated H^p the interval is within ~1.5x of the true spectral width, against ~50x for Gershgorin at k=16384, which
 * saves SP2 18 of 56 squarings.  m matrix-vector products of 8 k^2 bytes, all on the device.
 * Hp: device, k x k, read only.  eps_min / eps_max: HOST doubles.  Use through RFOE_OPT_LANCZOS_STEPS (rfoe_expand then
 * computes these bounds itself) or pass the result as RFOE_OPT_EPS_MIN / _MAX. */
int rfoe_bounds_lanczos(rfoe_handle_t h, const double* Hp, int64_t k, int m, double* eps_min, double* eps_max,
                        rfoe_stream_t stream);

/* The expansion.  Hp: device, k x k, bitwise symmetric, never written.  P: device, k x k, overwritten
 * with the final iterate (bitwise symmetric); must not overlap Hp.  0 < nocc < k.  tol: threshold of
 * the active stop rule (finite, >= 0).  Steps: Gershgorin bounds (or the override / Lanczos option) -> X_0 =
 * (eps_max I - H^p)/(eps_max - eps_min) -> recursion, each step taking the sign whose resulting trace (known beforehand
 * from Tr X_n and Tr X_n^2 = ||X_n||_F^2) lands nearer N_occ (for a spectrum inside [0,1] this is
 * "X^2 iff Tr X_n > N_occ", reading R4) -> P, tr(P H^p).  SP2_ACCEL additionally requires
 * eps_min <= RFOE_OPT_HOMO < RFOE_OPT_LUMO <= eps_max (else INVALID_ARG: the scaling factors would leave (0, 2)).
 * Returns OK, NOT_CONVERGED (P and stats still valid) or an error (P unspecified). */
int rfoe_expand(rfoe_handle_t h, const double* Hp, int64_t k, int64_t nocc, int variant, double tol, double* P,
                rfoe_stream_t stream);

/* Same as rfoe_expand with HOST buffers: copies Hp host->device, expands, copies P device->host
 * (staging buffers owned by the handle, sized for k_max).  Hp_host / P_host may be pageable or pinned. */
int rfoe_expand_host(rfoe_handle_t h, const double* Hp_host, int64_t k, int64_t nocc, int variant, double tol,
                     double* P_host, rfoe_stream_t stream);

/* One recursion step exposed on its own (kernel-level tests and roofline timing):
 * Xout = c2 * (X X) + c1 * X + c0 * I for a bitwise-symmetric device matrix X (k x k), computed by the
 * symmetric squaring kernel (upper-triangle tiles + mirror).  X and Xout must not overlap.
 * scalars (HOST, 5 doubles): Tr Xout, ||Xout||_F^2, ||X X - X||_F^2, Tr(X X), sum_ij (X X)_ij X_ij.
 * kernel_ms (HOST, may be null): CUDA-event time of the squaring kernel alone (padding copies excluded). */
int rfoe_square(rfoe_handle_t h, const double* X, int64_t k, double c2, double c1, double c0, double* Xout,
                double* scalars, float* kernel_ms, rfoe_stream_t stream);

/* The same step with the reduced-precision product of the mixed variant: X is split into
 * 11-bit (scaled FP16) parts X = Xh + Xl and X X is taken as Xh Xh + Xh Xl + Xl Xh on the tcgen05 tensor cores with FP32
 * accumulation (about FP32 accuracy); the update, mirror and the five scalars are FP64 as in rfoe_square.
 * kernel_ms covers the split pass and the product kernel.  Contract: |X_ij - (Tr X / k) delta_ij| < 2 (true for every
 * iterate of an expansion, whose spectrum lies in [0,1]); larger entries are clamped. */
int rfoe_square_reduced(rfoe_handle_t h, const double* X, int64_t k, double c2, double c1, double c0, double* Xout,
                        double* scalars, float* kernel_ms, rfoe_stream_t stream);

/* Issue-rate ceiling of the FP64 tensor pipe, measured on this device now: every SM runs 8 warps of a register-only
 * mma.m8n8k4.f64 (SASS DMMA.8x8x4) loop with 32 independent accumulators per warp -- the squaring kernel's inner loop with
 * its shared-memory loads removed -- for about `ms` milliseconds (1..10000); *tflops = issued flops / CUDA-event time.
 * No memory traffic, so this is the denominator the squaring's roofline fraction is quoted against (bench.py
 * `roofline.peak_measured`); it moves with the SM clock the device holds under this load.  tflops: HOST double. */
int rfoe_probe_fp64_peak(rfoe_handle_t h, double ms, double* tflops, rfoe_stream_t stream);

/* Symmetric product for commuting symmetric A, B (k x k, device): Cout = c2 * (A B) + c1 * A + c0 * I, upper
 * triangle computed and mirrored (the McWeeny step uses it with A = X^2, B = X).  scalars as in rfoe_square
 * with X replaced by A in the last three. */
int rfoe_symm_product(rfoe_handle_t h, const double* A, const double* B, int64_t k, double c2, double c1, double c0,
                      double* Cout, double* scalars, float* kernel_ms, rfoe_stream_t stream);

/* ---- steps either side of the expansion (sec. I, sec. III.A) -------------------
 * The paper's setting: the M x M Kohn-Sham matrix H "is orthogonally projected onto a carefully constructed
 * subspace ... (Rayleigh-Ritz step)", the resulting k x k H^p goes through the expansion above, which
 * "approximate[s] the density matrix in the subspace".  Neither step is printed in the paper; both are taken by
 * their plain definitions (reading R-RR) for a basis stored ONE STATE PER ROW:
 *   Psi, HPsi, Y : device, k x M row-major FP64 with row pitch ld (ldy for Y) >= M doubles; ld even and the
 *                  base 16-byte aligned (TMA pitch rule); 1 <= k <= k_max, 1 <= M <= 2^30 (rfoe_apply: M < 8.3e6).
 *   Psi rows are the (orthonormal) subspace basis, row j of HPsi is H applied to state j (formed matrix-free by
 *   the caller; H itself is never dense).  M need not be a multiple of anything: ragged tails are zero-filled. */

/* Rayleigh-Ritz projection: Hp_ij = sum_m Psi_im HPsi_jm for i <= j, mirrored to j > i (exactly symmetric for a
 * symmetric H; the mirror makes it bitwise symmetric, which rfoe_expand requires).  FP64 tensor cores, upper
 * tiles only, the sum over M split into slices added in a fixed order (bitwise reproducible).
 * Hp: device, k x k, ld = k, overwritten.  scalars (HOST, 2 doubles, may be null): Tr Hp, ||Hp||_F^2.
 * kernel_ms (HOST, may be null): CUDA-event time of the product + slice reduction. */
int rfoe_project(rfoe_handle_t h, const double* Psi, const double* HPsi, int64_t k, int64_t M, int64_t ld, double* Hp,
                 double* scalars, float* kernel_ms, rfoe_stream_t stream);

/* The subspace density matrix applied to the basis: Y = P Psi (Y_im = sum_j P_ij Psi_jm), and, when rho is not
 * null, the diagonal of the full-space density matrix Psi^T P Psi: rho_m = sum_i Psi_im Y_im (device, M doubles;
 * sum_m rho_m = Tr P = N_occ for an orthonormal basis).  P: device, k x k, ld = k (any k; it is copied into a
 * padded work matrix of the handle).  Y must not overlap Psi.  kernel_ms: the product kernel alone. */
int rfoe_apply(rfoe_handle_t h, const double* P, const double* Psi, int64_t k, int64_t M, int64_t ld, double* Y,
               int64_t ldy, double* rho, float* kernel_ms, rfoe_stream_t stream);

/* ---- many independent problems on ONE GPU (k-points, spins) --------------------------------------------------
 * One expansion of a mid-size H^p leaves part of the chip idle (k=2048: 136 tiles on 148 SMs, an epilogue and a
 * synchronisation per step), but independent problems can run side by side: n_handles handles, each with its own stream
 * and its own host thread (std::thread inside the library), take the n_problems problems from a shared counter in order.
 * Every problem goes through the rfoe_expand path of its handle.  With more than one handle at work, problems of
 * 1024 < k <= 4096 take the launch-per-step sequence (as with RFOE_OPT_RESIDENT = 0), whose kernels overlap across handles
 * and fill each other's gaps -- persistent launches of one CTA per SM cannot overlap; k <= 1024 keeps the small persistent
 * kernel (one expansion after the other, each 3-6x faster than launch-per-step).  Each P is bitwise the P of a lone
 * rfoe_expand call on the same path.  Measured on one B200: k=256, 16 handles: 8040 expansions/s (one handle: 2410;
 * round 1's launch-per-step path: 3400 / 430); k=2048, 4 handles: 92 expansions/s = 35 TFLOP/s executed (one: 81).
 *   handles[i], streams[i] : n_handles distinct handles (same device; options as set per handle) and their streams
 *   Hp[j], P[j], k[j], nocc[j], tol[j] : problem j (device matrices as for rfoe_expand; k[j] <= k_max of every handle);
 *                            all Hp[j] must be complete before the call (it does not order itself after other streams)
 *   status[j] (HOST, may be null): the rfoe_expand status of problem j;  stats[j] (HOST, may be null): its statistics
 * Returns OK when every problem returned OK, otherwise the first status in problem order that is not OK
 * (NOT_CONVERGED included); INVALID_ARG for null / duplicate handles or negative counts.  Blocks until all are done. */
int rfoe_expand_many(const rfoe_handle_t* handles, const rfoe_stream_t* streams, int n_handles, int n_problems,
                     const double* const* Hp, const int64_t* k, const int64_t* nocc, int variant, const double* tol,
                     double* const* P, int* status, rfoe_stats_t* stats);

/* ---- one expansion sharded over several GPUs (one process per GPU) -------------------------------------
 * The paper distributes the product over a process grid and communicates inside every multiplication
 * (PAPER.md:70-72).  Here every rank holds the whole X_n and squares a contiguous range of the upper-triangle
 * tile list (rfoe_shard_range); the exchange step is ONE all-gather per recursion step of this rank's new tiles
 * and their partial sums (4 n^2 (g-1)/g bytes received per GPU), after which every rank owns the whole X_{n+1}
 * and takes the same branch decision from the same sums in the same order: P is bitwise the single-GPU P.
 * Bounds, the affine map and the output pass are replicated on every rank (HBM-bound, O(k^2)).
 *
 * allgather(user, send, recv, bytes, stream): must gather `bytes` bytes from the DEVICE buffer `send` of every
 * rank into the DEVICE buffer `recv` (world x bytes, rank order), ordered after the work already enqueued on
 * `stream` and complete before work enqueued on `stream` afterwards (e.g. ncclAllGather on that stream, or
 * torch.distributed.all_gather_into_tensor under that current stream).  Returns 0 on success.
 * Every rank must call with the same H^p, k, nocc, variant, tol and options.  Variants: SP2, SP2_ACCEL and TRUNC;
 * others -> UNSUPPORTED. */
typedef int (*rfoe_allgather_fn)(void* user, const void* send, void* recv, int64_t bytes, rfoe_stream_t stream);
int rfoe_expand_sharded(rfoe_handle_t h, const double* Hp, int64_t k, int64_t nocc, int variant, double tol, double* P,
                        int rank, int world, rfoe_allgather_fn allgather, void* user, rfoe_stream_t stream);

/* ---- the same sharded expansion with the exchange fused into the squaring kernel (peer memory) --------------
 * Instead of pack / all-gather / unpack, the epilogue of every tile stores the tile, its mirror and its partial
 * record directly into the X_{n+1} and record arrays of ALL ranks through peer-mapped pointers (NVLink P2P), so
 * the transfer is spread over the whole launch and overlaps the tensor-core work of the other tiles; the only
 * collective left per step is a barrier.  Setup, once per handle (all ranks created with the same k_max):
 *   same process (threads, tests):  rfoe_shard_local_ptrs on every handle, then rfoe_shard_set_peers(h, rank,
 *       world, ptrs) with ptrs[4 d .. 4 d + 3] = rank d's four pointers (peer access enabled by the caller);
 *   one process per GPU:            rfoe_shard_ipc_export -> all-gather the 4 x 64-byte handles -> 
 *       rfoe_shard_ipc_import(h, rank, world, handles of all ranks in rank order) (cudaIpcOpenMemHandle).
 * barrier(user, stream): must return after every rank's work enqueued on its stream so far has COMPLETED
 * (e.g. cudaStreamSynchronize + an MPI / torch.distributed barrier).  Returns 0 on success.
 * rfoe_expand_sharded_p2p calls barrier once on entry (before its first store into a peer: a rank still finishing the
 * previous expansion reads the same buffers) and once per recursion step; every rank must therefore make the same
 * sequence of calls with the same arguments, or the barrier never completes.
 * rfoe_shard_ipc_import checks every opened buffer with cudaDeviceCanAccessPeer and returns RFOE_ERR_NO_PEER_ACCESS (nothing
 * left mapped) when a peer cannot be reached; fall back to rfoe_expand_sharded then.
 * Variants and the bitwise-equality guarantee as for rfoe_expand_sharded. */
#define RFOE_IPC_HANDLE_BYTES 64
typedef int (*rfoe_barrier_fn)(void* user, rfoe_stream_t stream);
int rfoe_shard_local_ptrs(rfoe_handle_t h, void** ptrs /* 4 device pointers out: W0, W1, records of even / odd steps */);
int rfoe_shard_set_peers(rfoe_handle_t h, int rank, int world, void* const* ptrs /* 4 x world */);
int rfoe_shard_ipc_export(rfoe_handle_t h, void* handles /* 4 x RFOE_IPC_HANDLE_BYTES out */);
int rfoe_shard_ipc_import(rfoe_handle_t h, int rank, int world, const void* handles /* world x 4 x 64 bytes */);
int rfoe_expand_sharded_p2p(rfoe_handle_t h, const double* Hp, int64_t k, int64_t nocc, int variant, double tol, double* P,
                            rfoe_barrier_fn barrier, void* user, rfoe_stream_t stream);

/* Host-only helper (no device needed): the range [begin, begin + count) of the n_tiles upper-triangle tiles that
 * `rank` of `world` squares: ceil(n_tiles / world) tiles each, the last ranks possibly fewer (or none). */
int rfoe_shard_range(int64_t n_tiles, int rank, int world, int64_t* begin, int64_t* count);

/* Host-only introspection (no device needed): how one squaring at size k is launched on a GPU with sm_count SMs.
 * n_tiles upper-triangle 128 x 128 tiles; tiles [0, n_main) go to the main kernel in whole waves; the last
 * n_tiles - n_main tiles are cut into `slices` K-slices of kt_per_slice 16-wide chunks so that the otherwise nearly
 * empty last wave fills the SMs (slices = 1: no tail, plain launch).  DESIGN.md "Tail of a launch". */
int rfoe_plan_squaring(int64_t k, int sm_count, int64_t* n_tiles, int64_t* n_main, int* slices, int* kt_per_slice);

/* Host-only introspection (no device needed): how rfoe_expand runs the recursion of a k x k problem on a GPU with sm_count
 * SMs when RFOE_OPT_RESIDENT is on (variants SP2, SP2_ACCEL, TRUNC).  DESIGN.md section 13.
 *   path      0: one launch sequence per recursion step (k > 4096, or too few SMs)
 *             1 / 2: the whole recursion in one persistent launch of `grid` CTAs, one 32 x 32 (k <= 512) / 64 x 64
 *                (k <= 1024) output tile each with the whole contraction
 *             3: one persistent launch of `grid` CTAs sharing the n_tiles x kt chunk units (128 x 128 tile, 16-wide slice
 *                of the contraction) of a step in contiguous ranges of equal cost (stream-K)
 *   path 3 only: kt = chunks per tile; boundaries (grid + 1 ints, may be null): CTA b works on chunk units
 *             [boundaries[b], boundaries[b+1]) of the stream tile 0 chunks 0..kt-1, tile 1, ...; n_split = tiles not wholly
 *             inside one range, finished in the fix-up phase; split_tiles (3 ints per split tile, may be null; at most
 *             3 * grid + 3): tile, first CTA holding a segment of it, number of CTAs holding one. */
int rfoe_plan_resident(int64_t k, int sm_count, int* path, int* grid, int* kt, int64_t* n_tiles, int* n_split,
                       int* boundaries, int* split_tiles);

/* HOMO / LUMO estimates for A-Z-RFOE from the history of a finished Z-RFOE run (host only, no device needed).
 * The paper chooses the accelerated polynomials "based on HOMO ... and LUMO ... eigenvalues" and does not
 * say where they come from; in an SCF loop they come from the previous expansion (its refs. 31, 38; DESIGN.md reading
 * R-HL).  Every eigenvalue x of X_n obeys x (1 - x) <= e_n = ||X_n^2 - X_n||_F, so once the occupation is settled
 * (Tr X_n - Tr X_n^2 < 3/16 and |Tr X_n - N_occ| < 1/2, the McWeeny switch of reading R11) the image of the LUMO is
 * <= a_n = (1 - sqrt(1 - 4 e_n))/2 and the image of the HOMO is >= 1 - a_n.  Both are carried back through the inverses
 * of the steps taken ('S': sqrt(x), 'L': 1 - sqrt(1 - x), monotone) to X_0 and through the affine map to H^p; the
 * tightest pair over all admissible steps with e_n >= 1e-6 (below that, rounding in X_n shows) is returned:
 *     homo >= lambda_HOMO,  lumo <= lambda_LUMO  (up to rounding),   both inside the gap, typically within 1 % of it.
 * stats: the rfoe_stats_t of a plain SP2 run (FP64 steps only; any stop rule; also the sharded entry points).
 * Returns OK; UNSUPPORTED (other variant / reduced steps in the history); NOT_CONVERGED (no admissible step: run
 * stopped too early); INVALID_ARG.  Feed the result to RFOE_OPT_HOMO / RFOE_OPT_LUMO for the next SP2_ACCEL call. */
int rfoe_estimate_homo_lumo(const rfoe_stats_t* stats, double* homo, double* lumo);

int rfoe_set_option(rfoe_handle_t h, int key, double value); /* INVALID_ARG on bad value, UNSUPPORTED on bad key */
int rfoe_get_stats(rfoe_handle_t h, rfoe_stats_t* out);      /* copies the stats of the last call */
int rfoe_destroy(rfoe_handle_t h);                           /* frees everything the handle owns; h may be null */
const char* rfoe_strerror(int status);                       /* static string, never null */
int rfoe_version(void);                                      /* ABI version (major*100 + minor) */

#ifdef __cplusplus
}
#endif
#endif /* RFOE_H_ */
