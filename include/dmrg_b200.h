/* dmrg_b200.h -- C ABI of the B200-native DMRG hot path (arXiv:1309.5571).
 *
 * The path: the superblock projection  X' = H_SB X  inside the Davidson iteration
 * (Alg. 3).  With U(1) sectors the projection is the list of dense
 * block products
 *        X'_jl += c_alpha * A_{alpha,i->j} X_ik B_{alpha,k->l}^T        (Eq. 11)
 * over the operator pairs of the LR strategy (Eq. 9-10), plus the
 * BLAS-2 part of Alg. 3 (lines 3, 5, 12, 13; Alg. 4).
 *
 * Conventions
 *  - Every function returns int: 0 = DMRG_OK, >0 informational, <0 error.  No exception
 *    crosses the ABI; dmrg_last_error() gives the text of the last error of a handle
 *    (or of plan creation when the handle is NULL).
 *  - "DEVICE" pointers are CUDA device pointers owned by the caller; "HOST" pointers are
 *    host memory read (or written) during the call only.  The library never frees caller
 *    memory.  All device work is enqueued on the `cuda_stream` argument (a cudaStream_t
 *    passed as void*; NULL = the legacy default stream).
 *  - Flat superblock vector (readings A1, A5):
 *    the target sector is the concatenation, over the admissible sector pairs (i,k) with
 *    label(i) + label(k) == target sorted by (left sector index, right sector index), of
 *    the row-major d_i x d_k segment X_ik (left index slow, right index fast -- the
 *    memory order of the composite index of A (x) B).  dmrg_get_layout() reports it.
 *  - Operators are lists of dense row-major blocks A_{src->dst} of shape
 *    dims[dst] x dims[src].  The label shift of an operator is read off
 *    its blocks, never assumed (reading A4).
 *  - FP64 throughout.  Results are run-to-run bitwise reproducible: no floating-point
 *    atomics, every reduction has a fixed order (reading A23).
 *  - A plan serves ONE call at a time: its control words (ticket counter, ready counters),
 *    the T workspace, the split-K partial tiles, the X tile images and the Davidson state
 *    are per plan.  Calls on one plan must not be issued from several host threads at once.
 *    Calls may name different streams: the library orders them itself (every hot call
 *    records a plan-owned event, and a call on another stream first waits for it), so two
 *    applies of one plan never overlap on the device.  Use one plan per concurrent solve.
 *  - If a dependency wait inside the projection kernel ever gives up (seconds; a lost or
 *    foreign launch), a sticky error word is set and the next synchronising call returns
 *    DMRG_E_CUDA instead of hanging the stream.
 */
#ifndef DMRG_B200_H
#define DMRG_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ---- status codes ------------------------------------------------------------------ */
#define DMRG_OK               0
#define DMRG_NOT_CONVERGED    1   /* dmrg_lowest_eigenpair: max_iter applies spent        */
#define DMRG_E_INVALID_ARG   (-1)
#define DMRG_E_SECTOR        (-2) /* empty target space; block dims disagree with sector
                                     dims; blocks of one operator with different shifts  */
#define DMRG_E_ALLOC         (-3)
#define DMRG_E_CUDA          (-4)
#define DMRG_E_NUMERIC       (-5) /* NaN / zero norm (Davidson breakdown)                */

#define DMRG_HEISENBERG 1         /* PAPER.md:L43-54, Eq. 1-3                            */
#define DMRG_HUBBARD    2         /* PAPER.md:L66-82, Eq. 4-8 (spin-1/2)                 */

/* ---- problem statement ------------------------------------------------------------- */

/* Quantum-number sectors of one (enlarged) block. HOST arrays. */
typedef struct {
    int32_t        n_labels;   /* 1 = S_z (any integer unit); 2 = (N_up, N_dn)            */
    int32_t        n_sectors;
    const int32_t *labels;     /* HOST [n_sectors][n_labels]                              */
    const int32_t *dims;       /* HOST [n_sectors], >= 0 (0 = empty sector, skipped, A26) */
} dmrg_sectors;

/* One sector-blocked operator.  Index arrays HOST, data DEVICE. */
typedef struct {
    int32_t        n_blocks;   /* 0 = operator absent                                     */
    const int32_t *src;        /* HOST [n_blocks]: block b maps sector src[b] ...         */
    const int32_t *dst;        /* HOST [n_blocks]: ... to sector dst[b]                   */
    const int64_t *offset;     /* HOST [n_blocks]: element offset of block b in data      */
    const int32_t *ld;         /* HOST [n_blocks]: row stride (>= dims[src[b]]), row-major */
    const double  *data;       /* DEVICE                                                  */
} dmrg_block_op;

/* The superblock in the LR strategy.  Terms (reading A3):
 *  Heisenberg: H_L(x)I + I(x)H_R + J/2 (S+_L(x)S-_R + S-_L(x)S+_R) + J*Delta Sz_L(x)Sz_R
 *  Hubbard:    H_L(x)I + I(x)H_R - t sum_sigma [ (c+_L,s P_L)(x)c_R,s + (P_L c_L,s)(x)c+_R,s ]
 *              + U (D_L(x)I + I(x)D_R),  P_L = (-1)^{N_L} (reading A6: the fermion string of a
 *              right-block operator runs over the whole left block).
 *  S- and c are the transposes of the S+ and c+ blocks given here. */
typedef struct {
    int32_t       model;                      /* DMRG_HEISENBERG | DMRG_HUBBARD          */
    double        J, Delta, t, U;
    dmrg_sectors  left, right;
    dmrg_block_op H_L, H_R;                   /* block-diagonal, symmetric               */
    dmrg_block_op Sz_L, Sp_L, Sz_R, Sp_R;     /* Heisenberg boundary-site operators      */
    dmrg_block_op Cup_L, Cdn_L, Cup_R, Cdn_R; /* Hubbard c+_sigma of the boundary site,
                                                 strings inside the own block only       */
    dmrg_block_op D_L, D_R;                   /* optional sum_j n_up n_dn of the block;
                                                 folded into H_L/H_R at plan time (A7)   */
    const int32_t *target;                    /* HOST [n_labels]                         */
} dmrg_problem;

typedef struct {
    int32_t  k_max;     /* Davidson basis limit, 2..32 (PAPER.md:L271 uses 20)           */
    double   tol;       /* ||r||_2 <= tol, absolute (reading A17)                        */
    int32_t  max_iter;  /* cap on H applies in dmrg_lowest_eigenpair                     */
    int32_t  reorth;    /* classical Gram-Schmidt passes in lines 12-13: 1 or 2 (A16)    */
    uint64_t seed;      /* start vector seed when x0 == NULL                             */
    int32_t  tile;      /* projection tile selector: 0 = auto                            */
    int32_t  check_every; /* dmrg_lowest_eigenpair: host reads the device convergence flag
                             every this many iterations (0 = default 8)                   */
    int32_t  reserve_basis; /* != 0: allocate the drivers' own V, W at plan creation, so that
                               dmrg_lowest_eigenpair / dmrg_block_lowest_eigenpairs allocate nothing */
    int32_t  shard_rank, shard_count; /* output sharding over several GPUs: with
                             shard_count > 1 the plan projects only the output segments owned by shard_rank
                             (dmrg_get_shard); the other segments of y are left untouched.  0 = no sharding. */
    int32_t  max_rhs;     /* largest number of vectors one projection launch takes
                             (dmrg_apply_H_multi, block Davidson): 1..4, 0 = 1.  The per-apply
                             workspaces are allocated max_rhs times at plan creation.       */
} dmrg_options;

typedef struct {
    int64_t n;                 /* target-sector dimension                                 */
    int32_t n_pairs;           /* admissible sector pairs (segments)                      */
    int32_t n_records;         /* operation records                       */
    int32_t n_gemms;           /* dense GEMMs per apply (identity factors skipped)        */
    int64_t flop_per_apply;    /* algorithmic FLOP, reading A24                           */
    int64_t operator_elems;    /* operator-block elements the apply reads (unpadded)      */
    int64_t apply_bytes;       /* 8*(operator_elems + 2n): compulsory traffic per apply   */
    int32_t stage1_units, stage2_units; /* work units (64x64 tile x K slice) of the two GEMM
                                           stages; one persistent launch runs both          */
    int32_t stage2_split_tiles;/* output tiles whose concatenated K is split              */
    int64_t pool_bytes;        /* repacked operator pool                                  */
    int64_t workspace_bytes;   /* T + split-K partials + Davidson scratch                 */
    int64_t device_bytes;      /* everything the plan allocated on the device             */
    int32_t kernel_launches_per_apply;
    int32_t kernel_launches_per_step;  /* dmrg_davidson_step at reorth passes = options   */
    int64_t flop_stage1, flop_stage2;  /* split of flop_per_apply over the two GEMM stages */
    int64_t launches;                  /* kernels launched by the hot-path entry points of
                                          this plan since it was created (host-side count) */
} dmrg_stats;

/* The superblock in the l-1-1-r strategy (Eq. 12-13; Alg. 2):
 *   H_SB = sum_alpha A_alpha^(l) (x) a_alpha (x) b_alpha (x) B_alpha^(r)
 * for the spin-1/2 Heisenberg chain, expressed by the operators of the four subsystems: block l, site 1, site 2, block r.
 * The caller gives the UN-enlarged blocks: H (block-diagonal), Sz and S+ of the block's boundary site (the last site of l,
 * the first site of r), labels = 2 S_z (any integer unit in which S+ of a site shifts the label by +2; the sites carry
 * labels -1, +1).  Quadruplets (reading A35): H_l 1 1 1, 1 1 1 H_r, and for each of the three bonds l-site1, site1-site2,
 * site2-r the terms J/2 (S+ S- + S- S+) + J Delta Sz Sz.  Sector by sector these are Eq. 11 records on the block operators
 * themselves (largest matrix O(m^2) instead of O((2m)^2)), and the bond between the two sites needs no GEMM.
 * Flat vector (reading A36): left composite sectors (s, sigma1) at index 2 s + sigma1 (down = 0, up = 1), right composite
 * sectors (sigma2, s') at index sigma2 * n_r + s'; segments = admissible pairs sorted by (left, right) composite index, each
 * row-major d_l(s) x d_r(s').  dmrg_get_layout reports the composite indices. */
typedef struct {
    double        J, Delta;
    dmrg_sectors  left, right;             /* sectors of block l and block r (n_labels = 1)            */
    dmrg_block_op H_l, Sz_l, Sp_l;         /* H_l block-diagonal; Sz_l block-diagonal; S+_l shifts +2  */
    dmrg_block_op H_r, Sz_r, Sp_r;
    int32_t       target_twice_sz;
} dmrg_problem_l11r;

typedef struct dmrg_plan *dmrg_handle_t;

/* ---- plan -------------------------------------------------------------------------- */

/* Builds everything that is constant over the Davidson iterations ("A, B
 * are fixed"): admissible pairs, operation records grouped by output segment (L342, L358:
 * "all records of the same output on the same [owner]" -> atomics-free accumulation),
 * per-record association order by FLOP (A24), the repacked operator pool (scaled,
 * transposed, stored as 8 KB tile images), the work units of the grouped launch, diag(H_SB)
 * (A14) and all workspaces.  Reads the operator data on the device (stream NULL) and
 * synchronises before returning.  opts may be NULL (k_max 20, tol 1e-10, max_iter 2000,
 * reorth 1).  On failure *out = NULL and dmrg_last_error(NULL) has the reason. */
int dmrg_plan_create(const dmrg_problem *problem, const dmrg_options *opts, dmrg_handle_t *out);
/* Same, for the l-1-1-r strategy; every other entry point (dmrg_apply_H, the Davidson calls, ...) works on the handle. */
int dmrg_plan_create_l11r(const dmrg_problem_l11r *problem, const dmrg_options *opts, dmrg_handle_t *out);
int dmrg_plan_destroy(dmrg_handle_t h);

/* Flat-vector layout.  Any output pointer may be NULL.  left_sector/right_sector/seg_offset
 * are HOST arrays of n_pairs entries (call once with NULL arrays to get n_pairs). */
int dmrg_get_layout(dmrg_handle_t h, int64_t *n, int32_t *n_pairs,
                    int32_t *left_sector, int32_t *right_sector, int64_t *seg_offset);
int dmrg_get_stats(dmrg_handle_t h, dmrg_stats *stats);
/* Output sharding ("all records of the same output on the same device", L362 workload per
 * output): longest-processing-time assignment of n_outputs outputs with the given costs to n_ranks ranks (descending cost,
 * ties by lower index; least loaded rank, ties by lower rank).  Host only, no device needed; every rank computes the same
 * table.  dmrg_get_shard reports the table a plan used: owner HOST [n_pairs] (all 0 without sharding). */
int dmrg_partition_outputs(int32_t n_outputs, const int64_t *cost, int32_t n_ranks, int32_t *owner);
int dmrg_get_shard(dmrg_handle_t h, int32_t *owner);
/* diag(H_SB) on the target sector (reading A14) copied to a DEVICE array of n doubles. */
int dmrg_get_diag(dmrg_handle_t h, double *d_out, void *cuda_stream);
const char *dmrg_last_error(dmrg_handle_t h);

/* ---- hot path ---------------------------------------------------------------------- */

/* y = H_SB x on the target sector: Eq. 11 over all records (Alg. 3 line 2).
 * x, y DEVICE, n doubles each, must not overlap; y is overwritten.  Asynchronous on the
 * stream; no allocation; one kernel launch (both GEMM stages of every record). */
int dmrg_apply_H(dmrg_handle_t h, const double *x, double *y, void *cuda_stream);

/* Starts a Davidson run (Alg. 3 "Require"): V(:,0) = x0/||x0||, k = 1,
 * B = 0.  V, W DEVICE, column-contiguous n x k_max with column stride ldv >= n doubles
 * (ldv even keeps 16-byte vector loads).  x0 DEVICE n doubles, or NULL for a seeded
 * N(0,1)-like start (options.seed; reading A19).  start_at_argmin_diag != 0 with
 * x0 == NULL selects the deterministic start e_argmin(D) (lowest index on ties). */
int dmrg_davidson_init(dmrg_handle_t h, const double *x0, int32_t start_at_argmin_diag,
                       double *V, double *W, int64_t ldv, void *cuda_stream);

/* One call of Alg. 3 (readings A13-A18):
 *   W(:,k-1) = H_SB V(:,k-1); B(0:k,k-1) = V^T W(:,k-1); (lambda,y) lowest eigenpair of B;
 *   x = V y; r = W y - lambda x; rho = ||r||; if rho <= tol -> converged;
 *   restart collapse when k == k_max (A15); t = r / g(lambda - D) (A14);
 *   reorth x { s = V^T t; t -= V s } (A16); V(:,k) = t/||t||; k += 1.
 * In: *k = number of orthonormal columns held in V (W(:,0..k-2) = H V(:,0..k-2), B as
 * left by the previous call).  Out: *k updated (k+1, or 2 after a restart; unchanged when
 * converged), *lambda, *resnorm, *converged (HOST).  Synchronises the stream once to read
 * these three numbers.  Returns DMRG_E_NUMERIC on breakdown (A18/step 9).
 * With lambda, resnorm and converged ALL NULL the step is only enqueued (no synchronisation,
 * the way dmrg_lowest_eigenpair runs its loop): *k is advanced as if the step did not
 * converge (the basis size is a host-known function of the step count), the convergence
 * test still runs on the device and every step enqueued after it fires is a no-op that
 * leaves V, W, B and the reported state untouched; read the state with dmrg_davidson_poll. */
int dmrg_davidson_step(dmrg_handle_t h, double *V, double *W, int64_t ldv, int32_t *k,
                       double *lambda, double *resnorm, int32_t *converged, void *cuda_stream);

/* dmrg_davidson_step without its line 2: W(:,k-1) = H_SB V(:,k-1) has been formed by the caller -- e.g. summed over the
 * ranks of an output-sharded projection (each rank applies its own plan to V(:,k-1), then one all-reduce) -- and lines 3-14
 * run as usual.  Same arguments and conventions as dmrg_davidson_step. */
int dmrg_davidson_step_given_w(dmrg_handle_t h, double *V, double *W, int64_t ldv, int32_t *k, double *lambda,
                               double *resnorm, int32_t *converged, void *cuda_stream);

/* dmrg_davidson_step for a caller that keeps (part of) the basis on the HOST -- the setting of the
 * paper's hybrid code, where each new basis vector is uploaded and H_SB x downloaded every
 * iteration (Alg. 7 lines 3 and 7, L432-445).  v_in_host (n doubles, or NULL) is copied into
 * V(:,k-1) on the stream before line 2; w_out_host (n doubles, or NULL) receives W(:,k-1) =
 * H_SB V(:,k-1), copied on a plan-owned side stream as soon as the projection has finished so
 * that the transfer overlaps lines 3-13 (on a restart step the collapse waits for it).  Pinned
 * host memory is needed for the copies to be asynchronous.  A PINNED v_in_host (cudaHostAlloc /
 * cudaHostRegister memory, anything cudaPointerGetAttributes reports as host memory) is not copied
 * by the copy engine at all: loader CTAs of the projection kernel read it over PCIe segment by
 * segment, in the order the work units need the segments, write V(:,k-1) and the operand images,
 * and the other CTAs start on the 16-row blocks that have arrived (same results bit for bit; a plan of
 * the l-1-1-r strategy and pageable memory take the plain copy).  Always synchronises (stream and
 * side stream) before returning; the other arguments and the return value are those of
 * dmrg_davidson_step.  If the run had already converged the step is a no-op and w_out_host
 * receives W(:,k-1) as it stands. */
int dmrg_davidson_step_host(dmrg_handle_t h, double *V, double *W, int64_t ldv, int32_t *k,
                            const double *v_in_host, double *w_out_host, double *lambda,
                            double *resnorm, int32_t *converged, void *cuda_stream);

/* Synchronises the stream and reports the state after the last EXECUTED (not no-op) step:
 * lambda, rho = ||r|| (Alg. 3 lines 4-7), converged flag, number of executed iterations
 * since dmrg_davidson_init (HOST; any may be NULL).  DMRG_E_NUMERIC on breakdown. */
int dmrg_davidson_poll(dmrg_handle_t h, double *lambda, double *resnorm, int32_t *converged,
                       int32_t *iters, void *cuda_stream);

/* Small-matrix state of the last step for lock-step tests: B (k_max x k_max, row-major)
 * and y (k_max) copied to HOST arrays (either may be NULL).  dmrg_set_small loads B
 * (e.g. to resume from a caller-kept state). */
int dmrg_get_small(dmrg_handle_t h, double *B_host, double *y_host, void *cuda_stream);
int dmrg_set_small(dmrg_handle_t h, const double *B_host, void *cuda_stream);

/* x_out = V y / ||V y|| with the y of the last step (Alg. 3 line 5/8). DEVICE n doubles. */
int dmrg_ritz_vector(dmrg_handle_t h, const double *V, int64_t ldv, int32_t k,
                     double *x_out, void *cuda_stream);

/* Driver (Alg. 3 looped): lowest eigenpair of H_SB on the target sector.
 * x0 DEVICE or NULL (seeded start; start_at_argmin_diag as in dmrg_davidson_init);
 * x_out DEVICE n doubles (normalised Ritz vector); lambda, resnorm, iters HOST.
 * Uses plan-owned V, W (2 * n * k_max doubles: allocated at plan creation with
 * options.reserve_basis != 0, else on the first call of a driver).  The convergence
 * test runs on the device; the host polls it every options.check_every iterations, so up
 * to check_every-1 no-op launches may follow convergence; the reported iteration count is
 * the exact one.  Returns DMRG_OK, DMRG_NOT_CONVERGED or an error. */
int dmrg_lowest_eigenpair(dmrg_handle_t h, const double *x0, int32_t start_at_argmin_diag,
                          double *x_out, double *lambda, double *resnorm, int32_t *iters,
                          void *cuda_stream);

/* ---- several vectors at once: block Davidson (Davidson-Liu) ------------ */

/* Y(:,r) = H_SB X(:,r), r < nrhs <= options.max_rhs, in ONE grouped launch (ticket = unit * nrhs + r).  x, y DEVICE,
 * column-contiguous with column strides ldx, ldy >= n; must not overlap.  Asynchronous, no allocation. */
int dmrg_apply_H_multi(dmrg_handle_t h, int32_t nrhs, const double *x, int64_t ldx, double *y, int64_t ldy,
                       void *cuda_stream);

/* Block iteration for the nb lowest eigenpairs (1 <= nb <= options.max_rhs, 2 nb <= k_max), the textbook method in
 * the line order of Alg. 3 with nb columns where Alg. 3 has one (readings A29-A32):
 *   init:  V(:,0..nb-1) = orthonormalised X0 (thin QR, positive diagonal); k = na = nb.   X0 DEVICE n x nb, stride ldx0.
 *   step:  W(:,new) = H_SB V(:,new) for the *na newest columns (one launch); G(:,new) = V^T W(:,new);
 *          (theta_i, y_i) the nb lowest eigenpairs of G; x_i = V y_i; r_i = W y_i - theta_i x_i;
 *          converged when every ||r_i|| <= tol; otherwise one correction t_i = r_i / g(theta_i - D) per pair that is NOT
 *          converged, restart (collapse to the nb Ritz vectors) when they would not fit, Gram-Schmidt against V
 *          (options.reorth passes) and among themselves, append.  *k and *na (number of appended columns, still to be
 *          projected) are updated; theta, resnorm: HOST arrays of nb.  Synchronises the stream.
 *   ritz:  X_out(:,i) = V y_i / ||V y_i|| with the y_i of the last step (k = basis size of that step).
 * V, W as in dmrg_davidson_init.  DMRG_E_NUMERIC: dependent or non-finite vectors. */
int dmrg_block_init(dmrg_handle_t h, int32_t nb, const double *X0, int64_t ldx0, double *V, double *W, int64_t ldv,
                    void *cuda_stream);
int dmrg_block_step(dmrg_handle_t h, double *V, double *W, int64_t ldv, int32_t *k, int32_t *na, int32_t nb,
                    double *theta, double *resnorm, int32_t *converged, void *cuda_stream);
int dmrg_block_ritz(dmrg_handle_t h, const double *V, const double *W, int64_t ldv, int32_t k, int32_t nb,
                    double *X_out, int64_t ldxo, void *cuda_stream);
/* Small-matrix state of the last block step: G (k_max x k_max, row-major) and Y (k_max x nb, row-major) to HOST. */
int dmrg_block_get_small(dmrg_handle_t h, int32_t nb, double *G_host, double *Y_host, void *cuda_stream);
/* Driver: the nb lowest eigenpairs from the start block X0 (DEVICE n x nb), on plan-owned V, W.  X_out DEVICE n x nb
 * (stride ldxo); theta, resnorm HOST nb; iters = block iterations, applies = projections of single vectors. */
int dmrg_block_lowest_eigenpairs(dmrg_handle_t h, int32_t nb, const double *X0, int64_t ldx0, double *X_out,
                                 int64_t ldxo, double *theta, double *resnorm, int32_t *iters, int32_t *applies,
                                 void *cuda_stream);

/* ---- the steps either side of the path: Alg. 1 lines 2, 5-7 ---- */

/* Line 5: reduced density matrix of one side of the plan's superblock from a target-sector vector x (DEVICE, n doubles,
 * normalised or not): side 0 = left, rho_i = sum_k X_ik X_ik^T; side 1 = right, rho_k = sum_i X_ik^T X_ik.
 * rho_out DEVICE: the sectors of that side in index order, each row-major d_s x d_s, back to back (sum_s d_s^2 doubles;
 * zero matrix for a sector without a pair).  Synchronises the stream. */
int dmrg_density_matrix(dmrg_handle_t h, const double *x, int32_t side, double *rho_out, void *cuda_stream);
/* Line 6: all eigenpairs of n_sectors symmetric blocks (layout as rho_out; rho is destroyed): U_out (same layout, columns =
 * eigenvectors by DESCENDING eigenvalue), w_out DEVICE (sum_s d_s doubles, descending per sector).  dims HOST. */
int dmrg_sector_eig(int32_t n_sectors, const int32_t *dims, double *rho, double *U_out, double *w_out, void *cuda_stream);
/* Line 7, the choice (host only): the m largest eigenvalues over all sectors (ties: lower sector index, then higher rank
 * inside the sector; eigenvalues <= 0 are never kept).  w_host as w_out; m_keep HOST [n_sectors] out; *discarded = sum of
 * all eigenvalues - sum of the kept ones. */
int dmrg_select_states(int32_t n_sectors, const int32_t *dims, const double *w_host, int32_t m, int32_t *m_keep,
                       double *discarded);
/* Line 7, the rotation: for every block b of `op` (index arrays HOST, data DEVICE), O'_b = U_dst(:, 0:m_dst)^T A_b
 * U_src(:, 0:m_src).  out_data DEVICE: the rotated blocks back to back, row-major m_dst x m_src (NULL: sizes only);
 * out_offset HOST [n_blocks]: element offset of each, -1 for a block that disappears; *out_elems: doubles needed. */
int dmrg_rotate_op(int32_t n_sectors, const int32_t *dims, const int32_t *m_keep, const double *U, const dmrg_block_op *op,
                   double *out_data, int64_t *out_offset, int64_t *out_elems, void *cuda_stream);

/* Alg. 1 looped (infinite-lattice algorithm) for the open spin-1/2 Heisenberg chain: from two single-site blocks,
 * every iteration enlarges both blocks by one site (line 2), finds the ground state of the LR superblock in the S_z = 0
 * sector with dmrg_lowest_eigenpair (line 3, start e_argmin(D)), builds both density matrices (5), diagonalises them (6) and
 * keeps the m_keep states of largest weight (7), until the superblock has n_sites sites.  One record per iteration (HOST
 * arrays of max_records; any may be NULL): superblock sites, ground-state energy, discarded weights, target-sector
 * dimension, Davidson iterations. */
typedef struct {
    int32_t n_sites;   /* even, >= 4 */
    int32_t m_keep;    /* block states kept after each iteration (the paper's m) */
    double  J, Delta;
    double  tol;       /* Davidson ||r|| <= tol (0 = 1e-10) */
    int32_t k_max;     /* Davidson basis limit (0 = 20) */
    int32_t max_iter;  /* Davidson applies per superblock (0 = 4000) */
} dmrg_idmrg_options;
int dmrg_infinite_heisenberg(const dmrg_idmrg_options *opts, int32_t max_records, int32_t *n_records, int32_t *n_sites,
                             double *energy, double *discarded_left, double *discarded_right, int64_t *target_dim,
                             int32_t *davidson_iters, void *cuda_stream);

/* ---- the Davidson BLAS-2 kernels on their own (Alg. 3 lines 3, 5-6, 12-13; Alg. 4) --- */

/* out[0..k) = V(:,0..k)^T w   (gemv_trans).  out DEVICE k doubles. */
int dmrg_gemv_trans(dmrg_handle_t h, const double *V, int64_t ldv, int32_t k,
                    const double *w, double *out, void *cuda_stream);
/* dmrg_gemv_trans for callers that may not allocate (code under CUDA stream capture, tight serving loops, harnesses that forbid
 * cudaMalloc): out[0..k) = V(:,0..k)^T w with NO plan handle and NO allocation of any kind -- the call makes no cudaMalloc,
 * cudaFree or allocating library call; it enqueues one 4-byte memset and one kernel on the stream.  Same kernel and arithmetic as
 * dmrg_gemv_trans (Alg. 3 lines 3 and 12; Alg. 4); the cross-CTA scratch of that kernel (one row of partial
 * sums per CTA, fixed-order final sum by the last CTA, and its arrival counter) lives in a file-scope device array of
 * DMRG_STATIC_SCRATCH_BYTES bytes that every GPU which loads the library holds until the process exits.
 *   V    DEVICE, column j at V + j*ldv, n doubles each (ldv >= n);   w  DEVICE, n doubles;   out  DEVICE, k doubles, overwritten.
 *   Limits: 1 <= k <= DMRG_STATIC_MAX_K, 1 <= n <= DMRG_STATIC_MAX_N; anything beyond is DMRG_E_INVALID_ARG with a message
 *   (dmrg_last_error(NULL)), nothing is launched.  The grid is at most 1024 CTAs (the rows of the scratch), so n does not size it.
 *   The current device is used; asynchronous on `cuda_stream`; V, w, out are the caller's and are not retained.
 *   ALL calls on a device share the one scratch array, which keeps the last call's contents (every call rewrites the partial sums
 *   it reads and clears the counter): calls that may OVERLAP on the GPU -- different streams without an ordering between them --
 *   race on it and give wrong results.  Calls on one stream, or ordered by events, are safe.  It does not interfere with plans. */
#define DMRG_STATIC_MAX_K 32
#define DMRG_STATIC_MAX_N (((int64_t)1) << 40)
#define DMRG_STATIC_SCRATCH_BYTES 278784
int dmrg_gemv_trans_static(const double *V, int64_t ldv, int64_t n, int32_t k, const double *w, double *out,
                           void *cuda_stream);
/* t -= V(:,0..k) s  and  *nrm2_out = ||t||^2 (gemv). s, nrm2_out DEVICE. */
int dmrg_gemv_sub(dmrg_handle_t h, const double *V, int64_t ldv, int32_t k,
                  const double *s, double *t, double *nrm2_out, void *cuda_stream);

/* ---- measurement helpers ----------------------------------------------------------- */

/* Register-only issue-rate probes used as the FP64 roofline denominator (MEASURED_PEAKS.json
 * has no FP64 entry): kind 0 = DFMA, 1 = DMMA.8x8x4 (mma.sync m8n8k4 f64).  Runs `reps`
 * launches on the stream, returns the best TFLOP/s in *tflops (HOST). */
int dmrg_probe_fp64_peak(int32_t kind, int32_t reps, double *tflops, void *cuda_stream);
/* Streams `bytes` of device memory (read-only sum) and returns GB/s (HOST). */
int dmrg_probe_hbm_read(int64_t bytes, int32_t reps, double *gbs, void *cuda_stream);
/* Per-kernel device time of the last dmrg_davidson_step when timing was enabled with
 * dmrg_set_timing(h, 1): ms[0] the apply (one grouped launch), [1] 0 (kept for layout), [2] V^T w, [3] small eig,
 * [4] residual+precondition, [5] restart collapse (0 unless k == k_max), [6] orthogonalise
 * (all passes), [7] normalise/append.  HOST array of 8. */
int dmrg_set_timing(dmrg_handle_t h, int32_t enable);
int dmrg_get_timing(dmrg_handle_t h, double *ms8);

/* Diagnostics: per-work-unit timeline of the LAST dmrg_apply_H of this plan, recorded only when the
 * plan was created with the environment variable DMRG_TRACE set (otherwise *n_units = 0).
 * trace_host: HOST array of 4 * max_units uint64 -- per unit, in issue (ticket) order:
 * start ns, end-of-main-loop ns, end ns (%globaltimer), packed word (bits 0-15 SM id, 16-31
 * k-tiles, 32-47 CTA, 48 stage-1 unit, 49 split-K unit, 50 wrote C); after the units, one
 * row per CTA: kernel entry, X images written, producer released, exit.  Synchronises the device. */
int dmrg_get_unit_trace(dmrg_handle_t h, uint64_t *trace_host, int32_t max_units, int32_t *n_units);

int dmrg_version(void);

#ifdef __cplusplus
}
#endif
#endif /* DMRG_B200_H */
