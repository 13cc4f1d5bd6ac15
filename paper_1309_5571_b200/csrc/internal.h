// internal.h -- structures shared by the host planner and the sm_100a kernels.
// Not part of the ABI (include/dmrg_b200.h is).
#pragma once
#include <cstdint>
#include <map>
#include <string>
#include <tuple>
#include <vector>
#include <cuda_runtime.h>
#include "../../include/dmrg_b200.h"

namespace dmrg {

// ---- grouped GEMM descriptors (projection, Eq. 11; L340 operation records) ----
// Every product on the path is brought to the form  C(MxN) = sum_items P(MxK) * Q(KxN), all
// row-major: right-block factors are stored transposed (B^T) and left-block factors pre-scaled
// by the record coefficient at plan time (operators are constant over the iteration, L340).
enum Base : uint8_t { BASE_XP = 0, BASE_Y = 1, BASE_T = 2, BASE_POOL = 3, BASE_PART = 4, BASE_XQ = 5, BASE_COUNT = 6 };

// Operand storage.  Every operand of the grouped kernel is stored as TILE IMAGES: 8 KB blocks holding exactly what one
// k-tile of the kernel keeps in shared memory, XOR-swizzled so that the DMMA fragment loads are bank-conflict free, edges
// zero-padded.  One k-tile of an operand = one bulk copy (cp.async.bulk).
//   P operand (M x K): image [m-tile][k-tile] at  off + (mt * ceil(K/16) + kt) * IMG, element (r, c) of the 64 x 16 tile
//                      at img_p_index(r, c);
//   Q operand (K x N): image [n-tile][k-tile] at  off + (nt * ceil(K/16) + kt) * IMG, element (k, c) of the 16 x 64 tile
//                      at img_q_index(k, c).
// BASE_POOL: the repacked operators (written once per plan); BASE_T: the T blocks between the two GEMM stages (written by
// the stage-1 epilogues); BASE_XP / BASE_XQ: the input vector's segments as P images (X_ik as M x K = d_i x d_k) and as
// Q images (K x N = d_i x d_k), written by phase 0 of every apply (all CTAs) from the caller's row-major vector.
struct GemmItem {
    long long p_off, q_off;   // element offsets of the operands' first images in their bases
    int K;
    uint8_t p_base, q_base;
    uint8_t xdep;             // 1: `dep` is the ready counter of an X segment (waited on only when x is streamed in, XShare)
    uint8_t pad;
    int dep;                  // index of the ready counter this item waits on: a T block of this launch, or an X segment (-1: none)
    int dep_need;             // T: 8 x tiles of that block (one count per consumer warp); X: elements of the segment
};

// Phase 0 table, one entry per segment X_ik (d_i x d_k, row-major at x + seg_off, ascending seg_off): where its P and Q images start
struct XSeg { long long seg_off, xp_off, xq_off; int di, dk; int rb0, pad; };     // rb0: first of the segment's row-block counters (streamed x)
// Streamed input (dmrg_davidson_step_host with pinned host memory): a few loader CTAs pull x over PCIe share by share, in
// the order the units need the segments, and publish the elements written per segment; the other CTAs start on the units.
struct XShare { int seg, lo, hi, pad; };   // elements [lo, hi) of segment `seg`
// Row blocks: 16 consecutive rows of a segment X_ik (= one k-tile of its Q images, a quarter of a tile row of its P images); the
// loaders count the elements written per row block (xrb), and a unit waits for exactly the row blocks its next stage reads.
struct XStream { const XShare *shares; int n_shares, n_loaders; double *x_copy; int *xrb; int n_xrb;
                 const int2 *xrows; int n_xrows; };      // xrows: (segment, first row) of every 8-row slab of x (phase 0)

struct GemmUnit {
    long long c_off;          // C(0,0) in its base
    long long part_off;       // first split-K partial slot of this tile (elements, BASE_PART)
    int ldc, M, N;            // whole output matrix
    int m0, n0;               // tile origin
    int item_begin, item_count;
    int kt_begin, kt_count;   // range in the flattened k-tile sequence of the tile's items
    int tile_id;              // split-K counter index (-1: not split)
    int split_idx, n_split;
    uint8_t c_base, c_vec2;
    uint8_t c_kind;           // C_ROWMAJOR (caller vector) | C_IMG_P | C_IMG_Q (T block, stored as the images stage 2 loads)
    uint8_t reducer;          // split-K: this slice (the tile's last in ticket order) sums the parked partials and writes C
    int signal;               // T-block ready counter to bump once this tile of T is written (-1: none)
    int cost;                 // scheduling weight (DMMA count + per-k-tile overhead)
    int item0, k00;           // where kt_begin falls: item index inside the unit's item list and k offset inside that item
    int axpy_begin, axpy_count;   // l-1-1-r: scaled copies of input segments added to this output (C_ROWMAJOR units only)
};

// l-1-1-r strategy: the bond between the two single sites maps a segment onto a segment of the same
// shape with a scalar -- no GEMM: y_seg += c * x[x_off ...] in the epilogue of the output tile.
struct AxpyItem { long long x_off; double c; };

// control words of one apply (device ints): ticket dispenser, finished count, X-image count, then one ready counter per T block
enum Ctrl : int { CTRL_TICKET = 0, CTRL_FINISHED = 1, CTRL_XREADY = 2, CTRL_XSHARE = 3, CTRL_DEP0 = 4 };   // XREADY: CTAs whose share of the X images is written

struct BasePtrs { double *p[BASE_COUNT]; };
// Several right-hand sides in ONE grouped launch (block Davidson): ticket = unit * nrhs + rhs; every
// per-apply buffer and counter set exists once per right-hand side, `stride` elements (or counters) apart.
constexpr int BMAX = 4;         // largest block size
struct RhsInfo { int nrhs, n_deps, n_counters, pad; long long stride[BASE_COUNT]; long long x_ld; };

// tile shape of the grouped kernel (gemm.cu is compiled for exactly these)
constexpr int BM = 64, BN = 64, BK = 16;
constexpr int IMG = BM * BK;    // doubles per tile image (P: 64 x 16, Q: 16 x 64)
#ifndef DMRG_CWARPS
#define DMRG_CWARPS 8
#endif
constexpr int CWARPS = DMRG_CWARPS;   // consumer warps per CTA of the grouped kernel; the ready counters count warps
enum CKind : uint8_t { C_ROWMAJOR = 0, C_IMG_P = 1, C_IMG_Q = 2 };
// 16-byte chunks of a row are XOR-ed with 2 * (row % 4): the 8 rows x 4 k (P) / 4 k x 8 columns (Q) of a DMMA fragment
// then fall on 32 distinct banks per half-warp.
__host__ __device__ inline int img_p_index(int r, int c) { return r * BK + ((((c >> 1) ^ (2 * (r & 3)))) << 1) + (c & 1); }
__host__ __device__ inline int img_q_index(int k, int c) { return k * BN + ((((c >> 1) ^ (2 * (k & 3)))) << 1) + (c & 1); }
inline long long img_p_elems(long long M, long long K) { return ((M + BM - 1) / BM) * ((K + BK - 1) / BK) * IMG; }
inline long long img_q_elems(long long K, long long N) { return ((N + BN - 1) / BN) * ((K + BK - 1) / BK) * IMG; }

// ---- plan-time device jobs ----
struct RepackJob {            // dst(rows x cols) = s1*op(src1) + s2*op(src2), op = transpose if flag; dst stored as images
    const double *src1, *src2;
    long long dst_off;
    int ld1, ld2, rows, cols;        // rows/cols of dst
    int transpose;
    int q_role;                      // 0: P images (rows = M, cols = K); 1: Q images (rows = K, cols = N)
    double s1, s2;
};
struct DiagJob {              // D_seg[a,b] += c * A(a,a) * B(b,b); null pointer = all ones
    long long seg_off;
    const double *da, *db;    // first image of the left (P role) / right (Q role) factor
    int ka, kb;               // their K (P: columns, Q: rows) -- fixes the image grid
    int rows, cols;
    double c;
};

// ---- Davidson device state (Alg. 3) ----
constexpr int KMAX = 32;
struct DavState {
    double B[KMAX * KMAX];    // row-major, kept symmetric (A18)
    double E[KMAX * KMAX];    // all eigenvectors of the last B (columns), warm start of the next small eig
    double y[KMAX];           // lowest eigenvector of B(0:k,0:k)
    double s[KMAX];           // Gram-Schmidt coefficients / scratch dot products
    double lambda, rho, rho2, tau2, nx2, x0n2;
    int done;                 // 1 once ||r|| <= tol
    int error;                // DMRG_E_NUMERIC sticky
    int iters;                // applies performed (stops counting once done)
    int k_used;               // basis size in the last executed step
    int sweeps;               // Jacobi sweeps of the last small eig
    int e_k;                  // size of the B whose eigenvectors E holds (0 = invalid)
    int gemm_error;           // sticky: a dependency wait of the grouped kernel gave up (lost / interleaved launch)
    int pad[1];
};

// ---- block Davidson device state (oracle/block_davidson.py)
struct BlockState {
    double G[KMAX * KMAX];       // V^T W, row-major, symmetric (the paper's B)
    double Y[KMAX * BMAX];       // Y[j * BMAX + r]: component j of the r-th lowest eigenvector of G(0:k,0:k)
    double S[KMAX * BMAX];       // S[r * KMAX + j]: dot products V(:,j)^T z_r of the last bvtw pass
    double theta[BMAX], rho2[BMAX], nx2[BMAX];
    double gram[BMAX * BMAX], Rinv[BMAX * BMAX];
    int error, pad[3];
};

struct Timing { bool enabled = false; cudaEvent_t ev[10]; double ms[8]; bool created = false; };

struct Plan {
    // problem (host copy)
    int model = 0; double J = 0, Delta = 0, t = 0, U = 0;
    int n_labels = 0;
    std::vector<int> labL, dimL, labR, dimR, target;
    dmrg_options opt{};
    // layout
    long long n = 0;
    std::vector<int> pairL, pairR;
    std::vector<long long> segOff;
    std::vector<int> owner;             // output sharding: rank that projects each output segment (all 0 without sharding)
    // device memory
    double *pool = nullptr, *tws = nullptr, *part = nullptr, *D = nullptr;
    double *ximg_p = nullptr, *ximg_q = nullptr;   // the input vector as P / Q tile images (rewritten by every apply)
    XSeg *xsegs = nullptr; int n_xsegs = 0;
    XShare *xshares = nullptr; int n_xshares = 0;   // streamed input: shares in the order of first use
    int *xrb = nullptr; int n_xrb = 0;              // streamed input: elements arrived per row block of every segment
    int2 *xrows = nullptr; int n_xrows = 0;         // (segment, first row) of every 8-row slab of x: one CTA each in scale_img_rows_kernel
    int n_deps_t = 0;                               // T-block counters; the X-segment counters follow (n_deps = n_deps_t + n_xsegs)
    const double *x_stream = nullptr;               // set for ONE apply_H: device-accessible (pinned host) source of x, streamed
    AxpyItem *axpy = nullptr; int axpy_count = 0;
    // the vector whose tile images are current because the library itself just wrote both (dmrg_davidson_step: line 14 writes
    // the appended vector and its images); consumed by the next projection of exactly that vector inside a step, cleared by
    // every other entry point that may see a different or modified vector
    const double *ximg_src = nullptr;
    int *counters = nullptr;
    GemmItem *items = nullptr;          // stage-1 items, then stage-2 items
    void *arena = nullptr;              // the ONE device allocation of the plan; every buffer below is a slice of it (plan.cu)
    std::vector<std::pair<void **, size_t>> arena_reqs;
    bool own_basis_in_arena = false;
    GemmUnit *units = nullptr;          // ticket order: stage-1 units, then stage-2 units
    GemmUnit *units_stream = nullptr;   // the same units in the ticket order of a streamed input (plan.cu)
    int n_units1 = 0, n_units2 = 0, n_deps = 0;
    int *ctrl = nullptr;                // Ctrl layout, self-resetting
    unsigned long long *trace = nullptr;   // optional per-unit timeline (4 words per unit), diagnostics
    int trace_units = 0;
    // Davidson scratch
    DavState *state = nullptr;          // device
    DavState *state_host = nullptr;     // pinned
    double *tvec = nullptr, *xs = nullptr, *ws = nullptr;   // n doubles each
    double *partials = nullptr;         // [vec_grid][KMAX+2]
    int *vec_counter = nullptr;
    int vec_grid = 0;
    double *Vown = nullptr, *Wown = nullptr; long long ldv_own = 0;   // dmrg_lowest_eigenpair
    // block Davidson (allocated at plan time when options.max_rhs >= 2)
    BlockState *bstate = nullptr, *bstate_host = nullptr;
    double *btvec = nullptr, *bxs = nullptr, *bws = nullptr, *bpartials = nullptr; long long bld = 0;
    // stats / misc
    dmrg_stats stats{};
    long long device_bytes = 0;
    long long launches = 0;             // hot-path kernel launches (host-side count)
    std::string err;
    Timing timing;
    int sm_count = 148;
    int max_rhs = 1;                    // right-hand sides the workspaces are sized for (options.max_rhs)
    long long tws_elems = 0, part_elems = 0, xp_elems = 0, xq_elems = 0; int n_counters = 0;   // per right-hand side
    // dmrg_davidson_step_host: W(:,k-1) leaves on a side stream as soon as the projection is done
    cudaStream_t side = nullptr;
    cudaEvent_t ev_apply = nullptr, ev_side = nullptr;
    // CUDA graphs of dmrg_davidson_step, one per (V, W, ldv, basis size)
    typedef std::tuple<const void *, const void *, long long, int> GraphKey;
    struct GraphEntry { cudaGraphExec_t exec; int k_next; int launches; const double *img_src; };
    std::map<GraphKey, GraphEntry> graphs;
    // one call at a time: a hot call on another stream than the previous one first waits for this event
    cudaEvent_t ev_last = nullptr; cudaStream_t last_stream = nullptr; bool last_valid = false;
    double *w_out_host = nullptr;       // non-null only while such a step is being enqueued
};

void set_global_error(const std::string &s);
int fail(Plan *p, int code, const std::string &msg);

// plan.cu
void partition_outputs(int n_outputs, const long long *cost, int n_ranks, int *owner);
int plan_build(const dmrg_problem *pr, const dmrg_options *opts, Plan **out, const dmrg_problem_l11r *l11 = nullptr);
void plan_free(Plan *p);

// plan.cu: ordering of hot calls of one plan across streams (include/dmrg_b200.h "A plan serves ONE call at a time")
void stream_enter(Plan *p, cudaStream_t st);
void stream_leave(Plan *p, cudaStream_t st);

// gemm.cu
cudaError_t gemm_kernel_setup();

// davidson.cu
void dav_setup(Plan *p);
int dav_init(Plan *p, const double *x0, int argmin_start, double *V, double *W, long long ldv, cudaStream_t st);
int dav_enqueue_step(Plan *p, double *V, double *W, long long ldv, int k, cudaStream_t st, int *k_next, bool skip_apply = false);
int dav_ritz(Plan *p, const double *V, long long ldv, int k, double *x_out, cudaStream_t st);
int dav_gemv_trans(Plan *p, const double *V, long long ldv, int k, const double *w, double *out, cudaStream_t st);
int dav_gemv_sub(Plan *p, const double *V, long long ldv, int k, const double *s, double *t, double *nrm2, cudaStream_t st);
// Optional side job of the last CTAs of an apply: pull the first `rows` rows of `cols` columns (column stride `ld`)
// into L2 for the kernel that follows (the Davidson basis for line 3), while the launch drains and HBM is idle.
struct Prefetch { const double *base = nullptr; long long ld = 0, rows = 0; int cols = 0, first_ticket = 0, n_ctas = 0; };
// davidson.cu: dmrg_gemv_trans_static (no plan, no allocation: scratch in a file-scope device array)
int dav_gemv_trans_static(const double *V, long long ldv, long long n, int k, const double *w, double *out, cudaStream_t st);
int apply_H(Plan *p, const double *x, double *y, const int *done_flag, cudaStream_t st, const Prefetch *pf = nullptr,
            int nrhs = 1, long long ldx = 0, long long ldy = 0, bool trust_images = false);

// block.cu
int block_alloc(Plan *p);
void block_free(Plan *p);
int bdav_init(Plan *p, int nb, const double *X0, long long ldx0, double *V, double *W, long long ldv, cudaStream_t st);
int bdav_step(Plan *p, double *V, double *W, long long ldv, int *k, int *na, int nb, double *theta, double *resnorm,
              int *converged, cudaStream_t st);
int bdav_ritz(Plan *p, const double *V, const double *W, long long ldv, int k, int nb, double *X_out, long long ldxo, cudaStream_t st);

// probe.cu
int probe_fp64(int kind, int reps, double *tflops, cudaStream_t st);
int probe_hbm(long long bytes, int reps, double *gbs, cudaStream_t st);

}  // namespace dmrg
