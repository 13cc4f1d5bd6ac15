// gemm.cu -- grouped FP64 tensor-core (DMMA) kernel of the projection.
//
// Computes, for every work unit, a 64x64 tile of  C = sum_items P_item * Q_item  (row-major
// operands, K concatenated over the unit's items) -- Eq. 11 of the paper,
//     X'_jl += A_{i->j} X_ik B_{k->l}^T
// with the sum over the records of one output realised as ONE long-K
// product so that nothing is accumulated through memory and no atomics are needed.
//
// sm_100a specifics: FP64 has no tcgen05/TMEM path (ptxas rejects .kind::f64); the FP64 tensor
// instruction is mma.sync m8n8k4 -> SASS DMMA.8x8x4, measured at 37.0 TFLOP/s on B200 (the
// DFMA pipe gives 33.9).  Operands are staged through shared memory with a 3-stage cp.async
// (LDGSTS) pipeline; padded rows (+4 doubles) make both fragment loads bank-conflict free.
// Ragged edges and odd row strides are handled by zero-filling cp.async (src-size < cp-size).
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

struct Cursor { int item; int k0; };   // position in the flattened k-tile sequence

struct ItemRegs {          // the current item, resolved once per item (not once per k-tile)
    const double *P, *Q;
    int ldp, ldq, K;
    bool pv, qv;
};
__device__ __forceinline__ ItemRegs resolve_item(const GemmItem *it, const BasePtrs &bases, bool xvec) {
    ItemRegs r;
    const long long po = it->p_off, qo = it->q_off;
    const int pb = it->p_base, qb = it->q_base;
    r.P = bases.p[pb] + po; r.Q = bases.p[qb] + qo;
    r.ldp = it->ldp; r.ldq = it->ldq; r.K = it->K;
    r.pv = it->p_vec2 && (pb != BASE_X || xvec);
    r.qv = it->q_vec2 && (qb != BASE_X || xvec);
    return r;
}

__device__ __forceinline__ void load_tiles(double *sP, double *sQ, const ItemRegs &it,
                                           int m0, int n0, int M, int N, int k0, int tid) {
    const double *P = it.P;
    const double *Q = it.Q;
    const int K = it.K;
    const bool pv = it.pv, qv = it.qv;
    // P tile: BM x BK
    if (pv) {
#pragma unroll
        for (int s = 0; s < (BM * BK / 2) / THREADS; s++) {
            int idx = tid + s * THREADS;
            int r = idx / (BK / 2), c = (idx % (BK / 2)) * 2;
            int valid = (m0 + r < M) ? min(max(K - (k0 + c), 0), 2) : 0;
            const double *src = valid ? P + (long long)(m0 + r) * it.ldp + k0 + c : P;
            cp_async16(sP + r * LDP + c, src, valid * 8);
        }
    } else {
#pragma unroll
        for (int s = 0; s < (BM * BK) / THREADS; s++) {
            int idx = tid + s * THREADS;
            int r = idx / BK, c = idx % BK;
            int valid = (m0 + r < M && k0 + c < K) ? 1 : 0;
            const double *src = valid ? P + (long long)(m0 + r) * it.ldp + k0 + c : P;
            cp_async8(sP + r * LDP + c, src, valid * 8);
        }
    }
    // Q tile: BK x BN
    if (qv) {
#pragma unroll
        for (int s = 0; s < (BK * BN / 2) / THREADS; s++) {
            int idx = tid + s * THREADS;
            int r = idx / (BN / 2), c = (idx % (BN / 2)) * 2;
            int valid = (k0 + r < K) ? min(max(N - (n0 + c), 0), 2) : 0;
            const double *src = valid ? Q + (long long)(k0 + r) * it.ldq + n0 + c : Q;
            cp_async16(sQ + r * LDQ + c, src, valid * 8);
        }
    } else {
#pragma unroll
        for (int s = 0; s < (BK * BN) / THREADS; s++) {
            int idx = tid + s * THREADS;
            int r = idx / BN, c = idx % BN;
            int valid = (k0 + r < K && n0 + c < N) ? 1 : 0;
            const double *src = valid ? Q + (long long)(k0 + r) * it.ldq + n0 + c : Q;
            cp_async8(sQ + r * LDQ + c, src, valid * 8);
        }
    }
}

// MODE 0: every DMMA of the 64x64x16 tile is issued (padding multiplies zeros);
// MODE 1: interior tiles take the same unpredicated path, edge tiles skip sub-tiles that hold only padding
//         (8-granular in M, N; 4-granular in K).
template <int STAGES, int MINB, int MODE>
__global__ void __launch_bounds__(THREADS, MINB)
grouped_gemm_kernel(const GemmUnit *__restrict__ units, const GemmItem *__restrict__ items, BasePtrs bases,
                    int *__restrict__ counters, const int *__restrict__ done_flag, int xvec, int yvec) {
    if (done_flag && *done_flag) return;
    extern __shared__ __align__(16) double smem[];
    double *sPbase = smem;
    double *sQbase = smem + STAGES * P_STAGE;
    __shared__ int s_is_last;

    const GemmUnit u = units[blockIdx.x];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm = (warp & 1) * 32, wn = (warp >> 1) * 32;
    const int g = lane >> 2, tg = lane & 3;
    const GemmItem *uitems = items + u.item_begin;

    double acc[4][4][2];
#pragma unroll
    for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < 4; j++) { acc[i][j][0] = 0.0; acc[i][j][1] = 0.0; }

    // producer cursor: walk to kt_begin; the consumer follows the same sequence STAGES-1 tiles behind
    Cursor pc{0, 0};
    {
        int skip = u.kt_begin;
        while (pc.item < u.item_count) {
            int nkt = (uitems[pc.item].K + BK - 1) / BK;
            if (skip < nkt) { pc.k0 = skip * BK; break; }
            skip -= nkt; pc.item++;
        }
    }
    const int KT = u.kt_count;
    ItemRegs cur{};
    if (KT > 0) cur = resolve_item(uitems + pc.item, bases, xvec != 0);
    Cursor cc = pc;
    int ccK = cur.K;
    auto produce = [&](int stage) {
        load_tiles(sPbase + stage * P_STAGE, sQbase + stage * Q_STAGE, cur, u.m0, u.n0, u.M, u.N, pc.k0, tid);
        pc.k0 += BK;
        if (pc.k0 >= cur.K) {
            pc.item++; pc.k0 = 0;
            if (pc.item < u.item_count) cur = resolve_item(uitems + pc.item, bases, xvec != 0);
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
        const int nk4 = (min(ccK - cc.k0, BK) + 3) >> 2;    // k4-steps with real K in this tile
        cc.k0 += BK;
        if (cc.k0 >= ccK) {
            cc.item++; cc.k0 = 0;
            if (cc.item < u.item_count) ccK = uitems[cc.item].K;
        }
        const double *pa = sPbase + (t % STAGES) * P_STAGE + (wm + g) * LDP + tg;
        const double *pb = sQbase + (t % STAGES) * Q_STAGE + tg * LDQ + wn + g;
        if (MODE == 0 || (full_warp_tile && nk4 == BK / 4)) {
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
        } else {
            for (int k4 = 0; k4 < nk4; k4++) {
                double a[4], b[4];
#pragma unroll
                for (int i = 0; i < 4; i++) a[i] = (i < mi) ? pa[i * 8 * LDP + k4 * 4] : 0.0;
#pragma unroll
                for (int j = 0; j < 4; j++) b[j] = (j < nj) ? pb[k4 * 4 * LDQ + j * 8] : 0.0;
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
    cp_async_wait<0>();

    double *C = bases.p[u.c_base] + u.c_off;
    const bool cvec = u.c_vec2 && (u.c_base != BASE_Y || yvec);
    if (u.n_split == 1) {
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
        return;
    }
    // split K: park the partial tile, the last unit of the tile to arrive sums all partials in
    // index order (deterministic whoever is last) and writes C.
    double *part = bases.p[BASE_PART] + u.part_off;
    {
        double *mine = part + (long long)u.split_idx * (BM * BN);
#pragma unroll
        for (int i = 0; i < 4; i++)
#pragma unroll
            for (int j = 0; j < 4; j++) {
                const int r = wm + i * 8 + g, c = wn + j * 8 + 2 * tg;
                __stcg(reinterpret_cast<double2 *>(mine + r * BN + c), make_double2(acc[i][j][0], acc[i][j][1]));
            }
    }
    __threadfence();
    __syncthreads();
    if (tid == 0) {
        int old = atomicAdd(&counters[u.tile_id], 1);
        s_is_last = (old == u.n_split - 1);
        if (s_is_last) counters[u.tile_id] = 0;   // self-cleaning for the next launch
    }
    __syncthreads();
    if (!s_is_last) return;
    __threadfence();
    for (int e = tid; e < BM * BN / 2; e += THREADS) {
        const int r = e / (BN / 2), c = (e % (BN / 2)) * 2;
        const int row = u.m0 + r, col = u.n0 + c;
        if (row >= u.M || col >= u.N) continue;
        double2 sum = make_double2(0.0, 0.0);
        for (int s = 0; s < u.n_split; s++) {
            double2 v = __ldcg(reinterpret_cast<const double2 *>(part + (long long)s * (BM * BN) + r * BN + c));
            sum.x += v.x; sum.y += v.y;
        }
        double *dst = C + (long long)row * u.ldc + col;
        if (cvec && col + 1 < u.N) *reinterpret_cast<double2 *>(dst) = sum;
        else { dst[0] = sum.x; if (col + 1 < u.N) dst[1] = sum.y; }
    }
}

}  // namespace

// kernel variants (selected once per process; DMRG_GEMM_VARIANT overrides the default for experiments)
typedef void (*gemm_fn)(const GemmUnit *, const GemmItem *, BasePtrs, int *, const int *, int, int);
struct Variant { const char *name; gemm_fn fn; int smem; };
static const Variant kVariants[] = {
    {"s3b4m0", grouped_gemm_kernel<3, 4, 0>, smem_bytes(3)},   // default: measured best at cfg3 / cfg5a
    {"s3b4m1", grouped_gemm_kernel<3, 4, 1>, smem_bytes(3)},
    {"s3b3m1", grouped_gemm_kernel<3, 3, 1>, smem_bytes(3)},
    {"s4b3m1", grouped_gemm_kernel<4, 3, 1>, smem_bytes(4)},
    {"s4b2m1", grouped_gemm_kernel<4, 2, 1>, smem_bytes(4)},
    {"s5b2m1", grouped_gemm_kernel<5, 2, 1>, smem_bytes(5)},
    {"s4b2m0", grouped_gemm_kernel<4, 2, 0>, smem_bytes(4)},
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

cudaError_t launch_grouped_gemm(const GemmUnit *units, int n_units, const GemmItem *items, const BasePtrs &bases,
                                int *counters, const int *done_flag, cudaStream_t st) {
    if (n_units <= 0) return cudaSuccess;
    const int xvec = ((reinterpret_cast<uintptr_t>(bases.p[BASE_X]) & 15) == 0) ? 1 : 0;
    const int yvec = ((reinterpret_cast<uintptr_t>(bases.p[BASE_Y]) & 15) == 0) ? 1 : 0;
    g_variant->fn<<<n_units, THREADS, g_variant->smem, st>>>(units, items, bases, counters, done_flag, xvec, yvec);
    return cudaGetLastError();
}

int apply_H(Plan *p, const double *x, double *y, const int *done_flag, cudaStream_t st) {
    BasePtrs b;
    b.p[BASE_X] = const_cast<double *>(x);
    b.p[BASE_Y] = y;
    b.p[BASE_T] = p->tws;
    b.p[BASE_POOL] = p->pool;
    b.p[BASE_PART] = p->part;
    cudaEvent_t *ev = p->timing.enabled ? p->timing.ev : nullptr;
    if (ev) cudaEventRecord(ev[0], st);
    p->launches += (p->n_units1 > 0 ? 1 : 0) + (p->n_units2 > 0 ? 1 : 0);
    cudaError_t e = launch_grouped_gemm(p->units1, p->n_units1, p->items1, b, p->counters, done_flag, st);
    if (ev) cudaEventRecord(ev[1], st);
    if (e == cudaSuccess) e = launch_grouped_gemm(p->units2, p->n_units2, p->items2, b, p->counters, done_flag, st);
    if (ev) cudaEventRecord(ev[2], st);
    if (e != cudaSuccess) return fail(p, DMRG_E_CUDA, std::string("apply_H launch: ") + cudaGetErrorString(e));
    return DMRG_OK;
}

}  // namespace dmrg
