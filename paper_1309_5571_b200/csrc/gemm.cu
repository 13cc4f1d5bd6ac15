// gemm.cu -- grouped FP64 tensor-core (DMMA) kernel of the projection: ONE launch per apply.
//
// Computes, for every work unit, a 64x64 tile of  C = sum_items P_item * Q_item  (row-major
// operands, K concatenated over the unit's items) -- Eq. 11 of the paper,
//     X'_jl += A_{i->j} X_ik B_{k->l}^T
// with the sum over the records of one output realised as ONE long-K
// product so that nothing is accumulated through memory and no atomics touch the data.
//
// Both stages of every record run in the same launch: units are handed out through a ticket
// counter in a fixed order -- all stage-1 units (T = X B^T or T = A X) first, then the stage-2
// units (X' tiles) -- and a stage-2 unit waits, item by item, on the "T block complete" counter of
// the stage-1 task that produces its operand.  A waiting unit only ever waits on units with a
// smaller ticket, which are running or finished, so the wait always ends.  This is the paper's
// "one stream per output, depth-first issue" (Alg. 7) without a launch boundary.
//
// sm_100a specifics: FP64 has no tcgen05/TMEM path (ptxas rejects .kind::f64); the FP64 tensor
// instruction is mma.sync m8n8k4 -> SASS DMMA.8x8x4, measured at 37.0 TFLOP/s on B200 (the
// DFMA pipe gives 33.9).  Operands are staged through shared memory with a 3-stage cp.async
// (LDGSTS) pipeline whose per-thread source pointers are bumped, not recomputed, per k-tile;
// padded rows (+4 doubles) make both fragment loads bank-conflict free.  Ragged edges and odd row
// strides are handled by zero-filling cp.async (src-size < cp-size); a warp whose 32x32 tile holds data only in
// its first 16 rows and/or columns runs a 2x4, 4x2 or 2x2 block of DMMA tiles instead of 4x4 (no predicates).
#include <cstdlib>
#include <string>
#include "internal.h"

namespace dmrg {

namespace {

constexpr int THREADS = 128;               // 4 warps, 2x2, warp tile 32x32
constexpr int LDP = BK + 4;                // 20 doubles: rows land on distinct bank groups
constexpr int LDQ = BN + 4;                // 68
constexpr int P_STAGE = BM * LDP;          // doubles
constexpr int Q_STAGE = BK * LDQ;
constexpr int smem_bytes(int stages) { return stages * (P_STAGE + Q_STAGE) * 8; }

__device__ __forceinline__ void cp_async16(void *smem, const void *g, int src_bytes) {
    unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(g), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async8(void *smem, const void *g, int src_bytes) {
    unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(s), "l"(g), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

__device__ __forceinline__ void dmma884(double &c0, double &c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
__device__ __forceinline__ int ld_acquire(const int *p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];\n" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned long long globaltimer() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %globaltimer;\n" : "=l"(t));
    return t;
}
__device__ __forceinline__ unsigned smid() {
    unsigned s;
    asm volatile("mov.u32 %0, %smid;\n" : "=r"(s));
    return s;
}


// Per-thread producer state of the current item: source pointers of this thread's first chunk in the
// P tile (BM x BK) and the Q tile (BK x BN), bumped by one k-tile after every produce.
//   16-byte mode: P chunk (row tid/8 + 16 s, col 2 (tid%8)), s < 4;  Q chunk (row tid/32 + 4 s, col 2 (tid%32)), s < 4
//    8-byte mode: P chunk (row tid/16 + 8 s, col tid%16),     s < 8;  Q chunk (row tid/64 + 2 s, col tid%64),     s < 8
struct Producer {
    const double *pP, *pQ;     // bumped
    const double *P0, *Q0;     // item bases (a legal address for zero-byte copies)
    int stepP, stepQ;          // element distance between consecutive s-chunks
    int K, k0;                 // item K; k0 of the next tile to produce
    bool pv, qv;
};

__device__ __forceinline__ void begin_item(Producer &pr, const GemmItem *it, double *const *bases, bool xvec,
                                           int m0, int n0, int k0, int tid, const int *ctrl) {
    const int dep = it->dep;
    if (dep >= 0) {            // operand is a T block of this launch: wait until all its tiles are written
        const int need = it->dep_need;
        const int *c = ctrl + CTRL_DEP0 + dep;
        while (ld_acquire(c) < need) __nanosleep(64);
    }
    const int pb = it->p_base, qb = it->q_base;
    pr.P0 = bases[pb] + it->p_off; pr.Q0 = bases[qb] + it->q_off;
    pr.K = it->K; pr.k0 = k0;
    pr.pv = it->p_vec2 && (pb != BASE_X || xvec);
    pr.qv = it->q_vec2 && (qb != BASE_X || xvec);
    const int ldp = it->ldp, ldq = it->ldq;
    if (pr.pv) { pr.pP = pr.P0 + (long long)(m0 + (tid >> 3)) * ldp + k0 + 2 * (tid & 7); pr.stepP = 16 * ldp; }
    else       { pr.pP = pr.P0 + (long long)(m0 + (tid >> 4)) * ldp + k0 + (tid & 15);    pr.stepP = 8 * ldp; }
    if (pr.qv) { pr.pQ = pr.Q0 + (long long)(k0 + (tid >> 5)) * ldq + n0 + 2 * (tid & 31); pr.stepQ = 4 * ldq; }
    else       { pr.pQ = pr.Q0 + (long long)(k0 + (tid >> 6)) * ldq + n0 + (tid & 63);     pr.stepQ = 2 * ldq; }
}

// rowmask16 / rowmask8: bit s set if this thread's s-th P chunk row is inside M (fixed per unit);
// colb16 / colb8: bytes of this thread's Q chunk that lie inside N (fixed per unit).
__device__ __forceinline__ void produce_tile(Producer &pr, double *sP, double *sQ, int tid,
                                             unsigned rowmask16, unsigned rowmask8, int colb16, int colb8) {
    const int K = pr.K, k0 = pr.k0;
    if (pr.pv) {
        const int kb = max(0, min(K - (k0 + 2 * (tid & 7)), 2)) * 8;
        double *d = sP + (tid >> 3) * LDP + 2 * (tid & 7);
#pragma unroll
        for (int s = 0; s < 4; s++) {
            const int bytes = ((rowmask16 >> s) & 1) ? kb : 0;
            cp_async16(d + s * 16 * LDP, bytes ? pr.pP + (long long)s * pr.stepP : pr.P0, bytes);
        }
    } else {
        const int kb = (k0 + (tid & 15) < K) ? 8 : 0;
        double *d = sP + (tid >> 4) * LDP + (tid & 15);
#pragma unroll
        for (int s = 0; s < 8; s++) {
            const int bytes = ((rowmask8 >> s) & 1) ? kb : 0;
            cp_async8(d + s * 8 * LDP, bytes ? pr.pP + (long long)s * pr.stepP : pr.P0, bytes);
        }
    }
    if (pr.qv) {
        double *d = sQ + (tid >> 5) * LDQ + 2 * (tid & 31);
        const int kr = K - k0 - (tid >> 5);          // rows left from this thread's first chunk row on
#pragma unroll
        for (int s = 0; s < 4; s++) {
            const int bytes = (4 * s < kr) ? colb16 : 0;
            cp_async16(d + s * 4 * LDQ, bytes ? pr.pQ + (long long)s * pr.stepQ : pr.Q0, bytes);
        }
        pr.pQ += 4 * (long long)pr.stepQ;            // BK rows = 4 steps of 4 rows
    } else {
        double *d = sQ + (tid >> 6) * LDQ + (tid & 63);
        const int kr = K - k0 - (tid >> 6);
#pragma unroll
        for (int s = 0; s < 8; s++) {
            const int bytes = (2 * s < kr) ? colb8 : 0;
            cp_async8(d + s * 2 * LDQ, bytes ? pr.pQ + (long long)s * pr.stepQ : pr.Q0, bytes);
        }
        pr.pQ += 8 * (long long)pr.stepQ;            // BK rows = 8 steps of 2 rows
    }
    pr.pP += BK;
    pr.k0 = k0 + BK;
}

// One k-tile of the warp tile restricted to its first MI x NJ sub-tiles (compile-time bounds: no predicates).
template <int MI, int NJ>
__device__ __forceinline__ void mma_ktile(double (&acc)[4][4][2], const double *pa, const double *pb) {
#pragma unroll
    for (int k4 = 0; k4 < BK / 4; k4++) {
        double a[MI], b[NJ];
#pragma unroll
        for (int i = 0; i < MI; i++) a[i] = pa[i * 8 * LDP + k4 * 4];
#pragma unroll
        for (int j = 0; j < NJ; j++) b[j] = pb[k4 * 4 * LDQ + j * 8];
#pragma unroll
        for (int i = 0; i < MI; i++)
#pragma unroll
            for (int j = 0; j < NJ; j++) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
    }
}

// MODE 0: every DMMA of the 64x64x16 tile is issued (padding multiplies zeros);
// MODE 1: sub-tiles that hold only padding are skipped (8-granular in M, N; 4-granular in K);
// MODE 2: warp tiles whose data fits in the first 2 sub-tile rows / columns run a 2x4, 4x2 or 2x2 DMMA block
//         (16-granular, no predicates), empty warp tiles run nothing.
template <int STAGES, int MINB, int MODE>
__global__ void __launch_bounds__(THREADS, MINB)
grouped_gemm_kernel(const GemmUnit *__restrict__ units, const GemmItem *__restrict__ items, BasePtrs bases,
                    int *__restrict__ counters, int *__restrict__ ctrl, int n_units, int n_deps,
                    const int *__restrict__ done_flag, int xvec, int yvec, unsigned long long *__restrict__ trace,
                    Prefetch pf) {
    if (done_flag && *done_flag) return;
    extern __shared__ __align__(16) double smem[];
    double *sPbase = smem;
    double *sQbase = smem + STAGES * P_STAGE;
    __shared__ int s_ticket, s_is_last;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_ticket = atomicAdd(&ctrl[CTRL_TICKET], 1);
    __syncthreads();
    const int ticket = s_ticket;
    // the unit descriptor lives in shared memory (read on demand) rather than in ~20 registers across the main loop
    __shared__ GemmUnit s_u;
    __shared__ double *s_base[BASE_COUNT];      // dynamically indexed: shared memory, not a local-memory copy of the parameter
    if (tid < (int)(sizeof(GemmUnit) / 4)) reinterpret_cast<int *>(&s_u)[tid] = reinterpret_cast<const int *>(units + ticket)[tid];
    if (tid == 32) { s_base[BASE_X] = bases.p[BASE_X]; s_base[BASE_Y] = bases.p[BASE_Y]; s_base[BASE_T] = bases.p[BASE_T]; s_base[BASE_POOL] = bases.p[BASE_POOL]; s_base[BASE_PART] = bases.p[BASE_PART]; }
    __syncthreads();
    const GemmUnit &u = s_u;
    unsigned long long t_start = 0, t_main = 0;
    if (trace && tid == 0) t_start = globaltimer();

    const int wm = (warp & 1) * 32, wn = (warp >> 1) * 32;
    const int g = lane >> 2, tg = lane & 3;
    const GemmItem *uitems = items + u.item_begin;

    double acc[4][4][2];
#pragma unroll
    for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < 4; j++) { acc[i][j][0] = 0.0; acc[i][j][1] = 0.0; }

    // per-unit constants of the producer
    unsigned rowmask16 = 0, rowmask8 = 0;
#pragma unroll
    for (int s = 0; s < 4; s++) if (u.m0 + (tid >> 3) + 16 * s < u.M) rowmask16 |= 1u << s;
#pragma unroll
    for (int s = 0; s < 8; s++) if (u.m0 + (tid >> 4) + 8 * s < u.M) rowmask8 |= 1u << s;
    const int colb16 = max(0, min(u.N - (u.n0 + 2 * (tid & 31)), 2)) * 8;
    const int colb8 = (u.n0 + (tid & 63) < u.N) ? 8 : 0;

    // producer cursor: walk to kt_begin; the consumer follows the same sequence STAGES-1 tiles behind
    int p_item = u.item0, p_k0 = u.k00;      // resolved by the planner
    const int KT = u.kt_count;
    Producer pr{};
    if (KT > 0) begin_item(pr, uitems + p_item, s_base, xvec != 0, u.m0, u.n0, p_k0, tid, ctrl);
    int c_item = p_item, c_k0 = p_k0, c_K = pr.K;
    auto produce = [&](int stage) {
        produce_tile(pr, sPbase + stage * P_STAGE, sQbase + stage * Q_STAGE, tid, rowmask16, rowmask8, colb16, colb8);
        if (pr.k0 >= pr.K) {
            p_item++;
            if (p_item < u.item_count) begin_item(pr, uitems + p_item, s_base, xvec != 0, u.m0, u.n0, 0, tid, ctrl);
        }
    };
    // sub-tiles of this warp that hold real rows / columns (8-granular): padding issues no DMMA
    const int mi = min(max(u.M - (u.m0 + wm) + 7, 0) >> 3, 4);
    const int nj = min(max(u.N - (u.n0 + wn) + 7, 0) >> 3, 4);
    const bool full_warp_tile = (mi == 4 && nj == 4);

    int issued = 0;
#pragma unroll
    for (int s = 0; s < STAGES - 1; s++) {
        if (issued < KT) { produce(s); issued++; }
        cp_async_commit();
    }
    for (int t = 0; t < KT; t++) {
        cp_async_wait<STAGES - 2>();
        __syncthreads();
        if (issued < KT) { produce(issued % STAGES); issued++; }
        cp_async_commit();
        const int nk4 = (min(c_K - c_k0, BK) + 3) >> 2;    // k4-steps with real K in this tile
        c_k0 += BK;
        if (c_k0 >= c_K) {
            c_item++; c_k0 = 0;
            if (c_item < u.item_count) c_K = uitems[c_item].K;
        }
        const double *pa = sPbase + (t % STAGES) * P_STAGE + (wm + g) * LDP + tg;
        const double *pb = sQbase + (t % STAGES) * Q_STAGE + tg * LDQ + wn + g;
        if (MODE == 2) {
            if (mi > 2 && nj > 2) mma_ktile<4, 4>(acc, pa, pb);
            else if (mi > 2 && nj > 0) mma_ktile<4, 2>(acc, pa, pb);
            else if (mi > 0 && nj > 2) mma_ktile<2, 4>(acc, pa, pb);
            else if (mi > 0 && nj > 0) mma_ktile<2, 2>(acc, pa, pb);
        } else if (MODE == 0 || (full_warp_tile && nk4 == BK / 4)) {
#pragma unroll
            for (int k4 = 0; k4 < BK / 4; k4++) {
                double a[4], b[4];
#pragma unroll
                for (int i = 0; i < 4; i++) a[i] = pa[i * 8 * LDP + k4 * 4];
#pragma unroll
                for (int j = 0; j < 4; j++) b[j] = pb[k4 * 4 * LDQ + j * 8];
#pragma unroll
                for (int i = 0; i < 4; i++)
#pragma unroll
                    for (int j = 0; j < 4; j++) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
            }
        } else if (mi > 0 && nj > 0) {
#pragma unroll
            for (int k4 = 0; k4 < BK / 4; k4++) {
                if (k4 < nk4) {
                    double a[4], b[4];
#pragma unroll
                    for (int i = 0; i < 4; i++) a[i] = pa[i * 8 * LDP + k4 * 4];
#pragma unroll
                    for (int j = 0; j < 4; j++) b[j] = pb[k4 * 4 * LDQ + j * 8];
#pragma unroll
                    for (int i = 0; i < 4; i++) {
                        if (i < mi) {
#pragma unroll
                            for (int j = 0; j < 4; j++)
                                if (j < nj) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
                        }
                    }
                }
            }
        }
    }
    cp_async_wait<0>();
    if (trace && tid == 0) t_main = globaltimer();

    bool writes_c = true;
    if (u.n_split > 1) {
        // split K: park the partial tile (fragment order: [slice][register pair][thread], coalesced 16-byte
        // stores); the last unit of the tile to arrive sums all slices IN SLICE ORDER (bitwise independent of
        // who is last, A22/A23) with the same thread <-> fragment mapping and writes C from registers.
        double2 *part = reinterpret_cast<double2 *>(s_base[BASE_PART] + u.part_off);
        double2 *mine = part + (long long)u.split_idx * (BM * BN / 2);
#pragma unroll
        for (int i = 0; i < 4; i++)
#pragma unroll
            for (int j = 0; j < 4; j++)
                __stcg(mine + (i * 4 + j) * THREADS + tid, make_double2(acc[i][j][0], acc[i][j][1]));
        __threadfence();
        __syncthreads();
        if (tid == 0) {
            const int old = atomicAdd(&counters[u.tile_id], 1);
            s_is_last = (old == u.n_split - 1);
            if (s_is_last) counters[u.tile_id] = 0;   // self-cleaning for the next launch
        }
        __syncthreads();
        writes_c = s_is_last != 0;
        if (writes_c) {
            __threadfence();
#pragma unroll
            for (int i = 0; i < 4; i++)
#pragma unroll
                for (int j = 0; j < 4; j++) { acc[i][j][0] = 0.0; acc[i][j][1] = 0.0; }
            for (int sl = 0; sl < u.n_split; sl++) {
                const double2 *src = part + (long long)sl * (BM * BN / 2) + tid;
#pragma unroll
                for (int h = 0; h < 2; h++) {          // 8 independent 16-byte loads in flight, twice
                    double2 v[8];
#pragma unroll
                    for (int q = 0; q < 8; q++) v[q] = __ldcg(src + (h * 8 + q) * THREADS);
#pragma unroll
                    for (int q = 0; q < 8; q++) {
                        acc[(h * 8 + q) >> 2][(h * 8 + q) & 3][0] += v[q].x;
                        acc[(h * 8 + q) >> 2][(h * 8 + q) & 3][1] += v[q].y;
                    }
                }
            }
        }
    }
    if (writes_c) {
        double *C = s_base[u.c_base] + u.c_off;
        const bool cvec = u.c_vec2 && (u.c_base != BASE_Y || yvec);
#pragma unroll
        for (int i = 0; i < 4; i++) {
            const int row = u.m0 + wm + i * 8 + g;
            if (row >= u.M) continue;
#pragma unroll
            for (int j = 0; j < 4; j++) {
                const int col = u.n0 + wn + j * 8 + 2 * tg;
                double *dst = C + (long long)row * u.ldc + col;
                if (cvec && col + 1 < u.N) {
                    *reinterpret_cast<double2 *>(dst) = make_double2(acc[i][j][0], acc[i][j][1]);
                } else {
                    if (col < u.N) dst[0] = acc[i][j][0];
                    if (col + 1 < u.N) dst[1] = acc[i][j][1];
                }
            }
        }
    }
    if (pf.base && ticket >= pf.first_ticket) {
        // side job of the last CTAs in ticket order (done when their unit is done: the launch is draining): L2 prefetch of one slice
        // of the rows the next kernel streams first; fire and forget, 128-byte lines
        const long long lines = (pf.rows + 15) >> 4;
        const int slice = ticket - pf.first_ticket;
        const long long l0 = lines * slice / pf.n_ctas, l1 = lines * (slice + 1) / pf.n_ctas;
        for (int c = 0; c < pf.cols; c++) {
            const double *col = pf.base + (long long)c * pf.ld;
            for (long long l = l0 + tid; l < l1; l += THREADS)
                asm volatile("prefetch.global.L2 [%0];" ::"l"(col + (l << 4)));
        }
    }
    // publish: this tile of a T block is complete (release: every thread's stores, then the counter);
    // units that publish nothing skip the fence
    if (writes_c && u.signal >= 0) __threadfence();
    __syncthreads();
    if (tid == 0) {
        if (writes_c && u.signal >= 0) atomicAdd(&ctrl[CTRL_DEP0 + u.signal], 1);
        if (trace) {
            unsigned long long *tr = trace + 4ull * ticket;
            tr[0] = t_start; tr[1] = t_main; tr[2] = globaltimer(); tr[3] = smid();
        }
        const int fin = atomicAdd(&ctrl[CTRL_FINISHED], 1);
        s_is_last = (fin == n_units - 1);
    }
    __syncthreads();
    if (s_is_last) {   // every other unit has finished: reset the control words for the next launch
        for (int e = tid; e < CTRL_DEP0 + n_deps; e += THREADS) ctrl[e] = 0;
    }
}

}  // namespace

// kernel variants (selected once per process; DMRG_GEMM_VARIANT overrides the default for experiments)
typedef void (*gemm_fn)(const GemmUnit *, const GemmItem *, BasePtrs, int *, int *, int, int, const int *, int, int,
                        unsigned long long *, Prefetch);
struct Variant { const char *name; gemm_fn fn; int smem; };
static const Variant kVariants[] = {
    {"s3b4m2", grouped_gemm_kernel<3, 4, 2>, smem_bytes(3)},   // default: measured best at cfg3 / 5a / 5b / 4096 sweep
    {"s3b4m0", grouped_gemm_kernel<3, 4, 0>, smem_bytes(3)},
    {"s3b4m1", grouped_gemm_kernel<3, 4, 1>, smem_bytes(3)},
    {"s4b3m2", grouped_gemm_kernel<4, 3, 2>, smem_bytes(4)},
};
static const Variant *g_variant = &kVariants[0];

cudaError_t gemm_kernel_setup() {
    if (const char *e = getenv("DMRG_GEMM_VARIANT"))
        for (const Variant &v : kVariants)
            if (std::string(v.name) == e) g_variant = &v;
    for (const Variant &v : kVariants) {
        cudaError_t err = cudaFuncSetAttribute(v.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, v.smem);
        if (err != cudaSuccess) return err;
    }
    return cudaSuccess;
}

int apply_H(Plan *p, const double *x, double *y, const int *done_flag, cudaStream_t st, const Prefetch *pf_in) {
    BasePtrs b;
    b.p[BASE_X] = const_cast<double *>(x);
    b.p[BASE_Y] = y;
    b.p[BASE_T] = p->tws;
    b.p[BASE_POOL] = p->pool;
    b.p[BASE_PART] = p->part;
    cudaEvent_t *ev = p->timing.enabled ? p->timing.ev : nullptr;
    if (ev) cudaEventRecord(ev[0], st);
    const int n_units = p->n_units1 + p->n_units2;
    p->launches += n_units > 0 ? 1 : 0;
    if (n_units > 0) {
        const int xvec = ((reinterpret_cast<uintptr_t>(x) & 15) == 0) ? 1 : 0;
        const int yvec = ((reinterpret_cast<uintptr_t>(y) & 15) == 0) ? 1 : 0;
        Prefetch pf;
        if (pf_in && pf_in->base && pf_in->cols > 0 && pf_in->rows > 0) {
            pf = *pf_in;
            pf.n_ctas = std::min(n_units, 4 * p->sm_count);
            pf.first_ticket = n_units - pf.n_ctas;
        }
        g_variant->fn<<<n_units, THREADS, g_variant->smem, st>>>(p->units, p->items, b, p->counters, p->ctrl, n_units,
                                                                 p->n_deps, done_flag, xvec, yvec, p->trace, pf);
    }
    if (ev) { cudaEventRecord(ev[1], st); cudaEventRecord(ev[2], st); }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(p, DMRG_E_CUDA, std::string("apply_H launch: ") + cudaGetErrorString(e));
    return DMRG_OK;
}

}  // namespace dmrg
