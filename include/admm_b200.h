/*
 * admm_b200.h -- C ABI of the B200-native batched ADMM solver for the Lightning-style
 * radiosurgery LP (arXiv 2509.08602).  One GPU, CUDA sm_100a.  No torch types, plain
 * pointers and sizes only.  Citations are PAPER.md line numbers (section / equation).
 *
 * The problem (App. A :308-344).  For plan p with class
 * weights w_k (dose units), beam-on-time weight w_BOT and an optional per-plan row mask:
 *
 *   P_p(t) = sum_k (w_k / N_{k,p}) sum_{i in class k, active in p} max(0, s_k (thr_k - Phi_i t))
 *            + w_BOT sum_j t_j ,   t >= 0
 *
 * solved through its dual  min c^T x, A x <= b, 0 <= x <= u  (Eq. 1, :47-49) by the ADMM
 * iteration Eq. (4b), (4c), (6), (7) (:70-94), all B plans at once (:96-98), one rho per
 * plan (:222), S = A A^T + I inverted once per handle and shared by every plan (:91).
 *
 * Threading: one handle is not thread-safe; distinct handles are independent.
 * Errors: every entry point returns a status; nothing throws or aborts across the ABI; on
 * error the outputs are untouched and admm_last_error() describes the failure.
 * There is no CPU fallback: without a CUDA sm_100 device every call fails with ADMM_ECUDA.
 */
#ifndef ADMM_B200_H
#define ADMM_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct admm_handle admm_handle;   /* opaque; one per (Phi, point classes) */

typedef enum {
    ADMM_OK = 0,
    ADMM_EINVAL = 1,    /* bad argument (null pointer, non-finite weight, B < 1, ...) */
    ADMM_ENOMEM = 2,    /* device or host allocation failed */
    ADMM_ECUDA = 3,     /* CUDA / cuBLAS / cuSOLVER error, or no sm_100 device */
    ADMM_ENOTSPD = 4,   /* Cholesky of S failed (cannot happen for finite Phi: lambda_min(S) >= 1) */
    ADMM_ESTATE = 5     /* call order violated (e.g. admm_get_state before any solve) */
} admm_status;

/* One dose-point class (Eq. 11-15 :314-326).
 * sense = +1: "dose >= threshold", under-dose is penalised (target surface / interior);
 * sense = -1: "dose <= threshold", over-dose is penalised (ring, low-dose volumes).
 * hard  = 2 : homogeneous hard class: u = infinity AND c = 0 -- the sector / isocenter coupling columns (-C_S^T ; T^T) of Eq. 12
 *             (:316, :330-332) given as rows of Phi: the primal constraint of such a row is sense * Phi_i t >= 0 (no threshold
 *             constant; threshold must be 1), e.g. tau_iso - sum_c t_(iso,s,c) / scale >= 0.  See admm_options.bot_rows.
 * hard  = 1 : u = infinity (organ-at-risk style hard constraint, Eq. 15 :322): the dual variable of such a point is clipped below
 *             only; in the primal, s (thr - Phi_i t) <= 0 is then a constraint instead of a penalty.  The class's weight is
 *             ignored and obj_out carries no term for it (whether the returned t satisfies the constraint to the accuracy reached
 *             is for the caller to check: the residual norms say how far the iteration is).  t = 0 must satisfy every hard class
 *             of sense -1; a hard class of sense +1 can make the LP infeasible (then the iteration does not converge). */
typedef struct {
    int32_t sense;
    float   threshold;
    int32_t hard;
} admm_class;

/* How Phi is stored in HBM and consumed by the tensor cores (BASELINE.json config 4). */
enum {
    ADMM_STORAGE_FP32_3XTF32 = 0, /* fp32 storage, hi/lo split on chip, 3 tf32 MMAs: the fp32 path (1e-4 parity) */
    ADMM_STORAGE_FP32_TF32   = 1, /* Phi rounded once to tf32 (kept in an fp32 container), 2 tf32 MMAs */
    ADMM_STORAGE_BF16        = 2, /* Phi rounded once to bf16 (half the HBM bytes), plan operands as bf16 hi/lo pairs, 2 bf16 MMAs (1e-2 parity) */
    ADMM_STORAGE_CSR         = 3  /* entries below csr_rel_threshold * max|Phi| dropped, CSR of Phi and of Phi^T, SpMM on the FP32 ALUs
                                     (kernel_path is ignored); S is formed from the thresholded matrix */
};

/* Which kernels run the two Phi contractions. */
enum {
    ADMM_PATH_TCGEN05 = 0,        /* tcgen05/TMEM/TMA kernels (the product path) */
    ADMM_PATH_SIMT    = 1         /* plain fp32 FFMA kernels: a slow on-device cross-check, same ABI.  They add the K terms of a product
                                     one after the other in fp32, so their error grows with N: 1e-4 iterate parity holds at the small sizes
                                     the tests use, not at n ~ 5000, N ~ 15000 (f5) */
};

typedef struct {
    int32_t storage;           /* ADMM_STORAGE_*                                                    */
    int32_t kernel_path;       /* ADMM_PATH_*                                                       */
    int32_t device;            /* CUDA device ordinal                                               */
    void*   stream;            /* cudaStream_t all work is enqueued on; NULL = the legacy default stream */
    int32_t check_every;       /* stopping rule tested every this many iterations; 0 => 10          */
    float   eps_abs;           /* absolute part of the stopping rule; 0 => 1e-6 (reading R7) */
    int32_t compaction;        /* must be 1: a plan that passes the stopping rule is frozen at that iterate and moved out of the
                                  active batch on the device (masking without compaction is not offered: 0 => ADMM_EINVAL) */
    float   csr_rel_threshold; /* ADMM_STORAGE_CSR only; 0 => 1e-3                                  */
    int32_t profile_kernels;   /* 1: CUDA events around every hot-path kernel (admm_get_kernel_times) */
    int32_t drain_kb;          /* the TMEM accumulator is drained into fp32 registers every this many 128-byte k-blocks
                                  (DESIGN.md section 7); 0 => default (1; 4 for bf16 storage), -1 => never        */
    int32_t k1_slab_kb;        /* K1 walks the point range in slabs of this many 32-point k-blocks so the slab of the plan
                                  operand stays in L2; 0 => chosen from the sizes            */
    int32_t presolve;          /* 1 (default): before iterating (tolerance mode only), plans whose box optimum x = argmin c^T x over
                                  [0,u] already satisfies A x <= b are settled in closed form: t = 0, iterations = 0, state = the
                                  ADMM fixed point (an LP presolve, not in the paper: DESIGN.md deviation D1); 0: every plan iterates */
    int32_t accum_debias;      /* the tensor core adds into its accumulator with truncation; optionally the drained sums are scaled back by the
                                  measured mean loss.  0: off (default), 100: on, other values > 0: percent of the
                                  measured factor */
    int32_t dose_only;         /* 1: the handle only serves admm_dose (II.C, :108-114: dose on a candidate grid between the passes): Phi is
                                  uploaded and tiled, S is neither formed nor factorised, admm_solve_batch is refused (ADMM_ESTATE) */
    float   warm_start_ratio;  /* > 0 (with presolve = 1, tolerance mode): a plan the presolve rejects whose box optimum violates A x <= b by at
                                  most this factor in every row ((A x_box)_j <= ratio * b_j) starts from the box state z1 = x_box,
                                  y1 = -c/rho, z2 = min(A x_box, b), y2 = A x_box - z2 instead of the zero iterate (deviation D3; the
                                  plans next to the presolve threshold of config 3 need 2.4x fewer iterations at ratio 2.5).  0 (default): zero start */
    const uint8_t* bot_rows;   /* HOST [n] 0/1 or NULL: the time variables whose row of A carries w_BOT in b (Eq. 13: b = (0, w_BOT): with
                                  the coupling blocks only the isocenter times do; P(t) then charges w_BOT * sum of THOSE t_j).  NULL =
                                  all n of them (the LP without coupling).  Read during admm_setup only. */
} admm_options;

/* Fills *opt with the defaults (3xTF32, tcgen05 path, device 0, default stream, check 10, 1e-6, compaction on, presolve on). */
void admm_default_options(admm_options* opt);

/*
 * Setup, steps S0-S2 of DESIGN.md ("compute its inverse just once and cache it",
 * :183/:213 row/column scaling).  Copies Phi into library-owned HBM (plus its transpose), builds
 * the preconditioner D_i = 1/N_class(i), R_j = 1/||row j of A D||_2, forms S = I + A^ A^^T in fp64,
 * Cholesky-factorises and inverts it in fp64.  Shared by every later admm_solve_batch.
 *
 *   phi            [N][ld] fp32 row-major, Phi[i][j] = dose rate at point i per unit of time variable j
 *                  (>= 0, finite).  Host pointer if phi_on_device == 0, else device pointer.
 *                  The caller keeps ownership; the library holds no reference after return.
 *   N, n, ld       points, time variables, row stride in elements (ld >= n)
 *   point_class    [N] HOST uint8, class id of each point, < n_classes
 *   classes        [n_classes] HOST, 1 <= n_classes <= 8
 *   opt            NULL => defaults
 * On success *out is a new handle (free with admm_destroy).
 */
admm_status admm_setup(admm_handle** out, const float* phi, int32_t phi_on_device,
                       int64_t N, int64_t n, int64_t ld,
                       const uint8_t* point_class, const admm_class* classes, int32_t n_classes,
                       const admm_options* opt);

/*
 * Solve B plans at once: steps H1-H6 of DESIGN.md = Eq. (6), (7), (4b), (4c) per iteration
 * (PAPER.md:73-94), stacked per :96, from the all-zero iterate.
 *
 *   weights     [B][n_classes+1] HOST fp32: w_class 0.., then w_BOT (config LP: 1, alpha, beta); >= 0, finite
 *   rho         [B] HOST fp32 step sizes (> 0), or NULL => (1/N_min) sqrt(w0/max(w_BOT, w0/65536)), w0 = 0.05, N_min = the
 *               smallest class count (the shape of Eq. 9, :219, scaled to the column scaling D; R8)
 *   row_mask    [B][ceil(N/32)] uint32 bit-packed (bit i%32 of word i/32 set => row i active in plan p;
 *               inactive rows get u = 0, :144), HOST or DEVICE pointer, or NULL => all rows active
 *   tol         relative tolerance of the stopping rule (R7); ignored if fixed_iters > 0
 *   max_iter    iteration cap (>= 1) when fixed_iters == 0
 *   fixed_iters > 0 => run exactly this many iterations for every plan, no masking, no compaction
 * Outputs (HOST or DEVICE pointers, detected; any may be NULL to skip):
 *   t_out       [B][n] fp32 beam-on times t_p = rho_p * R o y2_p (:80)
 *   obj_out     [B] fp64 primal objective P_p(t_p)
 *   res_out     [B][2] fp32 primal / dual residual norms ||x - z||, ||z+ - z|| at the plan's last tested iterate
 *   iters_out   [B] int32 iterations done (a multiple of check_every if the plan converged)
 * Synchronises opt->stream before returning.
 */
admm_status admm_solve_batch(admm_handle* h, int32_t B,
                             const float* weights, const float* rho, const uint32_t* row_mask,
                             float tol, int32_t max_iter, int32_t fixed_iters,
                             float* t_out, double* obj_out, float* res_out, int32_t* iters_out);

/*
 * Parity hook: the iterate of plan `plan` of the LAST admm_solve_batch in the paper's three-variable
 * form, recovered from the stored single state s = x + y (z = Pi(s), y = s - z):
 *   z1, y1 [N] fp32 ;  z2, y2 [n] fp64   (HOST or DEVICE pointers; any may be NULL)
 */
admm_status admm_get_state(admm_handle* h, int32_t plan, float* z1, float* y1, double* z2, double* y2);

/*
 * Test hook: ONE raw dose-rate contraction through the kernels of the selected path, no ADMM arithmetic.
 *   which = 0:  out[B][n] = small[B][N] . Phi      (the product of Eq. 6, before row scaling)
 *   which = 1:  out[B][N] = small[B][n] . Phi^T    (the product of Eq. 7)
 * small: HOST fp32 [B][K]; out: HOST fp64; 1 <= B <= 256.  Invalidates the state of the last solve.
 */
admm_status admm_contract_probe(admm_handle* h, int32_t which, int32_t B, const float* small, double* out);

/*
 * Dose calculation ("a weighted sum of precomputed kernels": one more batched Phi . T product) on the handle's
 * resident Phi, through the K3 contraction kernel of the selected path (passes of <= 96 plans on the fp32 path):
 *     dose_out[p][i] = Phi_i . t_p      for all N points of the handle and the B given time vectors.
 * It is what the two-pass optimisation of II.C (:108-114) needs between its passes: the first-pass dose of every plan on a grid of
 * candidate points, from which the plan's second-pass low-dose volume [D_LD, D_LD + Delta) is read off.  Works on any handle, also
 * one made with opt.dose_only = 1.
 *   t         [B][ld_t] fp32, HOST or DEVICE pointer (detected), ld_t >= n, finite
 *   dose_out  [B][N] fp32, HOST or DEVICE pointer (detected)
 * 1 <= B <= 496.  Invalidates the state of the last solve on this handle (admm_get_state then fails with ADMM_ESTATE).
 */
admm_status admm_dose(admm_handle* h, int32_t B, const float* t, int64_t ld_t, float* dose_out);

/*
 * Second-pass low-dose volumes (PAPER.md II.C.1, :110-114: "selecting a dose range around the low-dose threshold,
 * [D_LD, D_LD + Delta), and letting the low-dose volume be the portion of patient volume where the first-pass dose distribution is
 * within this range"), for all B plans at once, on the N points of the handle: admm_dose of the B time vectors, then
 *     bit i of in_volume[p] = ( d_lo <= dose_p[i] < d_hi )        (fp32 comparisons on the fp32 dose)
 *     bit i of any_volume   = OR over the plans                   (the union the second pass samples from, :144)
 * in the bit packing of admm_solve_batch's row_mask (bit i%32 of word i/32).
 *   t            [B][ld_t] fp32, HOST or DEVICE
 *   in_volume    [B][ceil(N/32)] uint32, HOST or DEVICE (detected)
 *   any_volume   [ceil(N/32)] uint32, HOST or DEVICE (detected), may be NULL
 *   dose_out     [B][N] fp32, HOST or DEVICE, may be NULL (the dose itself, as admm_dose returns it)
 * Same restrictions and side effects as admm_dose.
 */
admm_status admm_lowdose_volumes(admm_handle* h, int32_t B, const float* t, int64_t ld_t, float d_lo, float d_hi,
                                 uint32_t* in_volume, uint32_t* any_volume, float* dose_out);

/*
 * The dose-rate contraction of Eq. (6) (PAPER.md:89: W = G . Phi, all plans at once, :96) for callers that may not allocate: code
 * under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc.  No handle, no set-up call, and NO cudaMalloc / cudaFree
 * / allocating library routine in any call: the split-K partial sums and arrival counters live in one file-scope __device__ array of
 * ADMM_STATIC_SCRATCH_BYTES that every GPU which loads the library holds until the process exits.  Plain fp32 FFMA accumulation per
 * split (a variant of the ADMM_PATH_SIMT cross-check kernel, not the tcgen05 path), partial sums added in split order in fp64: the
 * same call gives the same bits every time.
 *     w_out[p][j] = sum_i g[p][i] * phi[i][j]
 *   phi     [N][ld] fp32 row-major, DEVICE pointer (the layout admm_setup takes), ld >= n
 *   g       [B][ld_g] fp32, DEVICE pointer, ld_g >= N
 *   w_out   [B][n] fp64, DEVICE pointer, dense
 *   device  CUDA device ordinal all three pointers belong to;  stream: cudaStream_t the work is enqueued on (NULL = legacy default)
 *   errbuf  HOST buffer of errbuf_len bytes that receives the message of a failed call (NUL-terminated), or NULL
 * Limit: B * n <= (ADMM_STATIC_SCRATCH_BYTES - 16384) / 4 = 2093056 outputs (e.g. 218 plans at n = 9600) and at most 4096 output
 * tiles of 64 x 64; beyond that the call fails with ADMM_EINVAL and touches nothing.  N is not limited.
 * Asynchronous: returns once the work is enqueued (one memset of the arrival counters, one kernel); it does not synchronise.
 * The first call on a device resolves the scratch array's address (cudaGetSymbolAddress, which loads the module): make it outside
 * stream capture.  Every call on a device shares the one array: calls that can overlap on the GPU (different streams, no ordering
 * between them) RACE on it -- order them.  Host threads may call concurrently as far as the library's own state goes.
 */
#define ADMM_STATIC_SCRATCH_BYTES (8 * 1024 * 1024)
admm_status admm_phit_apply_static(const float* phi, int64_t N, int64_t n, int64_t ld, const float* g, int64_t ld_g, int32_t B,
                                   double* w_out, int32_t device, void* stream, char* errbuf, int32_t errbuf_len);

/* Copies the preconditioner (fp64, HOST pointers, any may be NULL): D [N], R [n], Sinv [n][n]. */
admm_status admm_get_preconditioner(admm_handle* h, double* D, double* R, double* Sinv);

/*
 * Wall/device times of the last calls, milliseconds:
 *   ms[0] upload+transpose  ms[1] S = I + A^A^^T (syrk)  ms[2] Cholesky + inverse  ms[3] setup total
 *   ms[4] last solve: iterations (device)   ms[5] last solve: finalise (device)   ms[6] last solve total (host wall)
 *   ms[7] ADMM_STORAGE_CSR: density nnz / (N n) of the thresholded Phi, else 0
 *   plan_iters = sum over plans of iterations done in the last solve.
 */
admm_status admm_get_timing(admm_handle* h, double ms[8], int64_t* plan_iters);

/*
 * Per-kernel device time of the last solve when opt.profile_kernels = 1 (CUDA events on the
 * launching stream around every launch): for k in {0: K1 Phi^T.G, 1: K2 S^-1 apply, 2: K3 Phi.V + epilogue,
 * 3: convergence/compaction}: total_ms[k], launches[k].
 */
admm_status admm_get_kernel_times(admm_handle* h, double total_ms[4], int64_t launches[4]);

/* Number of kernels the library launched in the last solve (all of them its own). */
int64_t admm_last_launch_count(const admm_handle* h);

/* Message of the last error on this handle (or of the last failed admm_setup if h == NULL). Never NULL. */
const char* admm_last_error(const admm_handle* h);

void admm_destroy(admm_handle* h);

/* "paper_2509_08602_b200 <version> sm_100a" */
const char* admm_version(void);

#ifdef __cplusplus
}
#endif
#endif /* ADMM_B200_H */
