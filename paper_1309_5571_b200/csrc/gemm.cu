// gemm.cu -- grouped FP64 tensor-core (DMMA) kernel of the projection: ONE persistent launch per apply.
//
// Computes, for every work unit, a 64x64 tile of  C = sum_items P_item * Q_item  (K concatenated over the
// unit's items) -- Eq. 11 of the paper,
//     X'_jl += A_{i->j} X_ik B_{k->l}^T
// with the sum over the records of one output realised as ONE long-K product so that
// nothing is accumulated through memory and no atomics touch the data.
//
// Both stages of every record run in the same launch: units are handed out through a ticket counter in a
// fixed order -- all stage-1 units (T = X B^T or T = A X) first, then the stage-2 units (X' tiles) -- and a
// stage-2 unit waits, item by item, on the "T block complete" counter of the stage-1 task that produces its
// operand.  A waiting unit only ever waits on units with a smaller ticket, which are running or finished, so
// the wait always ends.  This is the paper's "one stream per output, depth-first issue" (Alg. 7,
// PAPER.md:L432-445) without a launch boundary.
//
// sm_100a specifics.  FP64 has no tcgen05/TMEM path (ptxas rejects .kind::f64); the FP64 tensor instruction is
// mma.sync m8n8k4 -> SASS DMMA.8x8x4 (one per 16 clocks per SM sub-partition: 37 TFLOP/s per chip).
// The kernel is WARP-SPECIALISED and PERSISTENT: each CTA = 8 consumer warps (8 of the tile's 64 8x8 accumulator
// sub-tiles each, in registers) + 1 producer warp, 2 CTAs per SM, a ring of STAGES stages of up to KPS = 3 consecutive k-tiles
// (a k-tile = 64x16 of P, 16x64 of Q; 48 KB per stage, two stages) with one "full" and one "empty" mbarrier per stage -- there
// is no CTA-wide barrier in the main loop.  Three k-tiles per barrier hand-over, executed as one straight-line stream of 96 DMMA
// per warp, is what lifts the core loop from 0.88 to 0.96 of the DMMA issue rate (measured in isolation): with one k-tile per
// stage every warp pays a try_wait, a header read, the address set-up and an arrive per 32 DMMA, and the compiler cannot carry
// fragment loads across the hand-over.
// Every operand (the repacked operator pool, the T workspace and -- after phase 0 of the kernel, in which all CTAs
// rewrite the caller's vector -- the input vector) is stored as 8 KB TILE IMAGES: the exact, bank-conflict-free (XOR-swizzled)
// shared-memory picture of one k-tile, edges zero-padded, so that a k-tile of an operand is staged by ONE bulk
// asynchronous copy of the TMA unit (cp.async.bulk, SASS UBLKCP) that signals the stage's mbarrier with complete_tx.
// One elected producer thread issues two such copies per stage (consecutive k-tiles of an operand are consecutive images); dependency waits are the producer's: the consumers
// keep draining the ring meanwhile.
#include <cstdlib>
#include <string>
#include "internal.h"

namespace dmrg {

namespace {

constexpr int CONSUMERS = CWARPS * 32;     // eight consumer warps, 8 of the tile's 64 accumulator sub-tiles each
constexpr int THREADS = CONSUMERS + 32;    // + 1 producer warp
static_assert(CWARPS == 8, "consumer layouts below are written for eight warps");
constexpr int KPS = 3;                     // k-tiles per ring stage (measured on the core loop alone: 1 -> 0.88-0.91 of the DMMA rate, 2 -> 0.94, 3 -> 0.96)
constexpr int STAGE_DOUBLES = 2 * KPS * IMG;   // up to KPS consecutive P images, then (at KPS * IMG) as many Q images: 48 KB
constexpr int UNIT_WORDS = (int)(sizeof(GemmUnit) / 4);
static_assert(UNIT_WORDS <= 32, "one lane per word of the unit descriptor");

enum : int { F_DATA = 1, F_LAST = 2, F_EXIT = 4, F_FIRST = 8, F_REDUCE = 16 };
constexpr int PUBLISH_DELAY = 1;           // a finished tile is fenced and signalled when the warp turns to its next stage (g + 1); a larger
                                           // value defers it by whole stages (measured: the waiting units lose what the fence costs here)
struct StageHdr {
    int flags, ticket, ext_m, ext_n;       // ext: rows / columns of the 64x64 tile that hold data
    int rot, layout, rhs, nk;              // sub-tile rotation and warp layout of the unit (see the consumers); right-hand side; k-tiles in the stage
    int u[UNIT_WORDS];                     // the unit descriptor (valid in the unit's last stage: epilogue)
};
constexpr int smem_bytes(int stages) { return stages * (STAGE_DOUBLES * 8 + (int)sizeof(StageHdr) + 16) + 128; }

// ---- PTX helpers
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(unsigned bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
// one 8 KB tile image, global -> shared, completion counted in bytes on the stage's mbarrier (TMA unit, UBLKCP)
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void *src, unsigned bytes, unsigned bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;\n" ::: "memory"); }
__device__ __forceinline__ bool mbar_test(unsigned bar, unsigned parity) {
    unsigned ok;
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "mbarrier.test_wait.parity.shared::cta.b64 P1, [%1], %2;\n"
        "selp.u32 %0, 1, 0, P1;\n"
        "}\n" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}

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

// ---------------------------------------------------------------- producer warp
struct Producer {
    const double *pP, *pQ;     // the next k-tile's images, bumped by one image per k-tile
    int K, k0;                 // item K; k0 of the next tile to produce
    int xq_di, xq_dk, xq_rb0;  // streamed x as the Q operand of the item (xq_dk > 0): its k-tiles are row blocks that arrive one by one
};

// Streamed x: waits until the row blocks [b0, b0 + nb) (nb <= 32) of a segment have arrived (one lane per row block).
__device__ __forceinline__ void wait_row_blocks(const int *xrb, int rb0, int di, int dk, int b0, int nb, int lane, int *err) {
    if (lane < nb) {
        const int b = b0 + lane;
        const int need = min(BK, di - b * BK) * dk;
        const int *c = xrb + rb0 + b;
        long long spins = 0;
        while (ld_acquire(c) < need) {
            __nanosleep(64);
            if (++spins > (1ll << 25)) { atomicExch(err, 1); break; }
        }
    }
    __syncwarp();
    fence_proxy_async();
}

__device__ __forceinline__ void begin_item(Producer &pr, const GemmItem *it, double *const *bases, const long long *stride,
                                           int rhs, int n_deps, int m0, int n0, int k0, int lane, const int *ctrl, int *err,
                                           int xmode, const XSeg *xsegs, const int *xrb) {
    pr.xq_dk = 0;
    if (it->xdep && xmode == 2) {
        // streamed x: as the P operand this tile reads rows m0 .. m0 + 63 of the segment (four row blocks, every k-tile: wait
        // here); as the Q operand its k-tiles ARE the row blocks, in the order of arrival: the stage loop waits for each group
        const XSeg sg = xsegs[it->dep];
        if (it->p_base == BASE_XP) wait_row_blocks(xrb, sg.rb0, sg.di, sg.dk, m0 / BK, (min(BM, sg.di - m0) + BK - 1) / BK, lane, err);
        else { pr.xq_di = sg.di; pr.xq_dk = sg.dk; pr.xq_rb0 = sg.rb0; }
    }
    const int dep = it->xdep ? -1 : it->dep;     // X segments: ready before the first unit unless x is streamed in (above)
    if (dep >= 0) {            // operand is a T block of this launch: wait until it is all written
        if (lane == 0) {
            const int need = it->dep_need;
            const int *c = ctrl + CTRL_DEP0 + rhs * n_deps + dep;
            long long spins = 0;
            while (ld_acquire(c) < need) {
                __nanosleep(32);
                if (++spins > (1ll << 26)) { atomicExch(err, 1); break; }   // seconds: a lost launch, not a slow one
            }
        }
        __syncwarp();
        fence_proxy_async();   // the T images were written through the generic proxy, the bulk copy reads through the async one
    }
    pr.K = it->K; pr.k0 = k0;
    const int KT = (pr.K + BK - 1) / BK;
    pr.pP = bases[it->p_base] + rhs * stride[it->p_base] + it->p_off + ((long long)(m0 / BM) * KT + k0 / BK) * IMG;
    pr.pQ = bases[it->q_base] + rhs * stride[it->q_base] + it->q_off + ((long long)(n0 / BN) * KT + k0 / BK) * IMG;
}

// ---------------------------------------------------------------- consumer warps
// The 64 x 64 tile is 8 x 8 sub-tiles of 8 x 8 (one DMMA.8x8x4 accumulator each); a warp owns a TH x TW block of them
// (TH * TW = 8 accumulator pairs, index i * TW + j) and the eight warps form a (8 / TH) x (8 / TW) grid.  Four layouts:
//   TH x TW = 4 x 2 (warp grid 2 x 4; full tiles: 6 fragment loads per 8 DMMA), 2 x 4, 8 x 1 and 1 x 8.
// For an EDGE tile (sm x sn sub-tiles with data) the producer picks the layout with the smallest busiest warp,
// min(TH, sm) * min(TW, sn): a CTA advances at the pace of its busiest warp, so e.g. a tile with 40 of 64 rows costs 5/8
// of a full tile with the 8 x 1 layout instead of 8/8 (cfg 3: -10 % on the critical path, cfg 5a: -16 %).
struct Lane {            // lane constants of the swizzled fragment addresses (internal.h: img_p_index / img_q_index)
    int offA[4];         // P: gq * BK + (((2 k4 + tg / 2) ^ 2 (gq % 4)) << 1) + tg % 2, per k4
    int rowB, c0, x2;    // Q: tg * BN + gq % 2;  gq / 2;  2 tg
};

// One k-tile of MI x NJ sub-tiles (compile-time bounds: no predicates); sc0 = first sub-tile column of the warp.
template <int MI, int NJ, int TW>
__device__ __forceinline__ void mma_ktile(double (&acc)[8][2], const double *sP, const double *sQ, const Lane &L, int sc0) {
    int ob[NJ];
#pragma unroll
    for (int j = 0; j < NJ; j++) ob[j] = L.rowB + (((((sc0 + j) << 2) | L.c0) ^ L.x2) << 1);
#pragma unroll
    for (int k4 = 0; k4 < BK / 4; k4++) {
        double a[MI], b[NJ];
#pragma unroll
        for (int i = 0; i < MI; i++) a[i] = sP[i * 8 * BK + L.offA[k4]];
#pragma unroll
        for (int j = 0; j < NJ; j++) b[j] = sQ[k4 * 4 * BN + ob[j]];
#pragma unroll
        for (int i = 0; i < MI; i++)
#pragma unroll
            for (int j = 0; j < NJ; j++) dmma884(acc[i * TW + j][0], acc[i * TW + j][1], a[i], b[j]);
    }
}
template <int TW, int NJ, int MI>
__device__ __forceinline__ void disp_mi(int mi, double (&acc)[8][2], const double *sP, const double *sQ, const Lane &L, int sc0) {
    if (mi == MI) mma_ktile<MI, NJ, TW>(acc, sP, sQ, L, sc0);
    else if constexpr (MI > 1) disp_mi<TW, NJ, MI - 1>(mi, acc, sP, sQ, L, sc0);
}
template <int TH, int TW, int NJ>
__device__ __forceinline__ void disp_nj(int mi, int nj, double (&acc)[8][2], const double *sP, const double *sQ, const Lane &L, int sc0) {
    if (nj == NJ) disp_mi<TW, NJ, TH>(mi, acc, sP, sQ, L, sc0);
    else if constexpr (NJ > 1) disp_nj<TH, TW, NJ - 1>(mi, nj, acc, sP, sQ, L, sc0);
}

// Epilogue of one warp: its TH x TW accumulator block -> C (row-major caller vector, or the tile images stage 2 loads).
// sr0 / sc0: first sub-tile row / column of the warp; gq, tg: DMMA fragment coordinates of the lane.
template <int TH, int TW>
__device__ __forceinline__ void store_c(double (&acc)[8][2], const GemmUnit &u, double *C, int sr0, int sc0, int gq, int tg, int yvec,
                                        const AxpyItem *__restrict__ axpy, const double *__restrict__ xr) {
    if (u.c_kind == C_ROWMAJOR) {
        const bool cvec = u.c_vec2 && (u.c_base != BASE_Y || yvec);
        // l-1-1-r: scaled copies of input segments of the same shape (the bond between the two sites)
        for (int q = 0; q < u.axpy_count; q++) {
            const AxpyItem it = axpy[u.axpy_begin + q];
            const double *xs = xr + it.x_off;
#pragma unroll
            for (int i = 0; i < TH; i++) {
                const int row = u.m0 + (sr0 + i) * 8 + gq;
                if (row >= u.M) continue;
#pragma unroll
                for (int j = 0; j < TW; j++) {
                    const int col = u.n0 + (sc0 + j) * 8 + 2 * tg;
                    if (col < u.N) acc[i * TW + j][0] = fma(it.c, xs[(long long)row * u.ldc + col], acc[i * TW + j][0]);
                    if (col + 1 < u.N) acc[i * TW + j][1] = fma(it.c, xs[(long long)row * u.ldc + col + 1], acc[i * TW + j][1]);
                }
            }
        }
#pragma unroll
        for (int i = 0; i < TH; i++) {
            const int row = u.m0 + (sr0 + i) * 8 + gq;
            if (row >= u.M) continue;
#pragma unroll
            for (int j = 0; j < TW; j++) {
                const int col = u.n0 + (sc0 + j) * 8 + 2 * tg;
                double *dst = C + (long long)row * u.ldc + col;
                if (cvec && col + 1 < u.N) {
                    *reinterpret_cast<double2 *>(dst) = make_double2(acc[i * TW + j][0], acc[i * TW + j][1]);
                } else {
                    if (col < u.N) dst[0] = acc[i * TW + j][0];
                    if (col + 1 < u.N) dst[1] = acc[i * TW + j][1];
                }
            }
        }
    } else if (u.c_kind == C_IMG_P) {
        // T (M x N) becomes the P operand of stage 2 (K = N): P images [m-tile][k-tile]; the column pair of an
        // accumulator is one 16-byte chunk (the pad column of an odd N receives the exact zero it computed)
        const int CT = (u.N + BK - 1) / BK;
        double *base = C + (long long)(u.m0 / BM) * CT * IMG;
#pragma unroll
        for (int i = 0; i < TH; i++) {
            const int r = (sr0 + i) * 8 + gq;
            if (u.m0 + r >= u.M) continue;
#pragma unroll
            for (int j = 0; j < TW; j++) {
                const int col = u.n0 + (sc0 + j) * 8 + 2 * tg;
                if (col < u.N)
                    *reinterpret_cast<double2 *>(base + (long long)(col / BK) * IMG + img_p_index(r, col % BK)) =
                        make_double2(acc[i * TW + j][0], acc[i * TW + j][1]);
            }
        }
    } else {
        // T (M x N) becomes the Q operand of stage 2 (K = M): Q images [n-tile][k-tile]
        const int CT = (u.M + BK - 1) / BK;
        double *base = C + (long long)(u.n0 / BN) * CT * IMG;
#pragma unroll
        for (int i = 0; i < TH; i++) {
            const int row = u.m0 + (sr0 + i) * 8 + gq;
            if (row >= u.M) continue;
#pragma unroll
            for (int j = 0; j < TW; j++) {
                const int c = (sc0 + j) * 8 + 2 * tg;
                if (u.n0 + c < u.N)
                    *reinterpret_cast<double2 *>(base + (long long)(row / BK) * IMG + img_q_index(row % BK, c)) =
                        make_double2(acc[i * TW + j][0], acc[i * TW + j][1]);
            }
        }
    }
}

// Phase 0: this CTA's contiguous share [lo, hi) of the caller's vector -> tile images (internal.h), written to the P images
// (X_ik as M x K) and to the Q images (X_ik as K x N) of the segment each element falls in.  Up to twelve independent loads per
// thread are in flight before the first store; scalar loads, any alignment of x.
__device__ __forceinline__ void ximg_share(const XSeg *__restrict__ segs, int n_segs, const double *__restrict__ x,
                                           long long lo, long long hi, double *__restrict__ xp, double *__restrict__ xq, int tid) {
    constexpr int U = 12;     // cfg 3 / 5a: a share is ~9-11 elements per thread -> every load of a share is in flight at once
    if (lo + tid >= hi) return;
    int a = 0;                                               // last segment with seg_off <= this thread's first element
    {
        int b = n_segs - 1;
        const long long e0 = lo + tid;
        while (a < b) { const int m = (a + b + 1) >> 1; if (segs[m].seg_off <= e0) a = m; else b = m - 1; }
    }
    XSeg sg = segs[a];
    long long next_off = (a + 1 < n_segs) ? segs[a + 1].seg_off : (long long)0x7fffffffffffffffll;
    for (long long base = lo + tid; base < hi; base += (long long)U * THREADS) {
        double v[U];
#pragma unroll
        for (int q = 0; q < U; q++) { const long long e = base + (long long)q * THREADS; v[q] = e < hi ? x[e] : 0.0; }
#pragma unroll
        for (int q = 0; q < U; q++) {
            const long long e = base + (long long)q * THREADS;
            if (e >= hi) break;
            while (e >= next_off) {                          // this thread's elements ascend: walk, do not search
                a++; sg = segs[a];
                next_off = (a + 1 < n_segs) ? segs[a + 1].seg_off : (long long)0x7fffffffffffffffll;
            }
            const int w = (int)(e - sg.seg_off), r = w / sg.dk, c = w - r * sg.dk;
            const int KTp = (sg.dk + BK - 1) / BK, KTq = (sg.di + BK - 1) / BK;
            xp[sg.xp_off + ((long long)(r / BM) * KTp + c / BK) * IMG + img_p_index(r % BM, c % BK)] = v[q];
            xq[sg.xq_off + ((long long)(c / BN) * KTq + r / BK) * IMG + img_q_index(r % BK, c % BN)] = v[q];
        }
    }
}

template <int STAGES, int MINB>
__global__ void __launch_bounds__(THREADS, MINB)
grouped_gemm_kernel(const GemmUnit *__restrict__ units, const GemmItem *__restrict__ items, BasePtrs bases,
                    int *__restrict__ counters, int *__restrict__ ctrl, int n_units, int n_deps,
                    const int *__restrict__ done_flag, int yvec, unsigned long long *__restrict__ trace,
                    Prefetch pf, int *__restrict__ err, const XSeg *__restrict__ xsegs, int n_xsegs,
                    const double *__restrict__ x, long long n, RhsInfo rh, int xmode, const AxpyItem *__restrict__ axpy,
                    XStream xs) {
    const int skip_phase0 = xmode != 0;      // xmode 0: phase 0 by all CTAs; 1: images are current; 2: streamed by loader CTAs
    if (done_flag && *done_flag) return;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double *stage_base = reinterpret_cast<double *>(smem_raw);
    StageHdr *hdrs = reinterpret_cast<StageHdr *>(smem_raw + (size_t)STAGES * STAGE_DOUBLES * 8);
    unsigned long long *bars = reinterpret_cast<unsigned long long *>(hdrs + STAGES);     // full[STAGES], empty[STAGES]
    __shared__ double *s_base[BASE_COUNT];      // dynamically indexed: shared memory, not a local-memory copy of the parameter
    __shared__ long long s_stride[BASE_COUNT];  // distance between the copies of a buffer for consecutive right-hand sides
    __shared__ int s_is_last;                   // end of the launch only

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; s++) {
            mbar_init(smem_u32(bars + s), 1);             // the producer's arrive(.expect_tx); the bytes complete the phase
            mbar_init(smem_u32(bars + STAGES + s), CWARPS);   // one arrival per consumer warp
        }
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    if (tid < BASE_COUNT) { s_base[tid] = bases.p[tid]; s_stride[tid] = rh.stride[tid]; }
    const int nrhs = rh.nrhs;
    unsigned long long *ctr = trace ? trace + 4ull * n_units * nrhs + 4ull * blockIdx.x : nullptr;   // per-CTA phase stamps (diagnostics)
    if (ctr && tid == 0) ctr[0] = globaltimer();
    // Phase 0: the caller's vector -> tile images (both operand roles), shared out over all CTAs; a CTA publishes its share
    // (CTRL_XREADY) and the producers wait for all shares before their first copy.  Every CTA of the grid is resident
    // (the grid is one wave), and each writes its share before it waits for anything.
    if (!skip_phase0) {        // (skipped when the caller has just written the images itself: scale_img_kernel, davidson.cu)
        const long long share = (n + gridDim.x - 1) / gridDim.x, lo = share * blockIdx.x;
        const XSeg *segs = xsegs;
        if ((size_t)n_xsegs * sizeof(XSeg) <= (size_t)STAGES * STAGE_DOUBLES * 8) {     // the segment table fits the (still idle) ring
            int *dst = reinterpret_cast<int *>(smem_raw);
            const int *src = reinterpret_cast<const int *>(xsegs);
            for (int e = tid; e < n_xsegs * (int)(sizeof(XSeg) / 4); e += THREADS) dst[e] = src[e];
            __syncthreads();
            segs = reinterpret_cast<const XSeg *>(smem_raw);
        }
        if (xs.xrows && segs != xsegs) {
            // one 8-row slab of a segment per CTA and trip, a warp per row, the lanes along the row: no search and no division per
            // element, coalesced loads (and Q-image stores); up to eight loads per lane in flight
            for (int sl = blockIdx.x; sl < xs.n_xrows; sl += gridDim.x) {
                const int2 rb = xs.xrows[sl];
                const XSeg sg = segs[rb.x];
                const int rr = rb.y + warp;
                if (warp >= 8 || rr >= sg.di) continue;
                const int dk = sg.dk;
                const int KTp = (dk + BK - 1) / BK, KTq = (sg.di + BK - 1) / BK;
                const long long row_off = sg.seg_off + (long long)rr * dk;
                const long long po = sg.xp_off + (long long)(rr / BM) * KTp * IMG, qo = sg.xq_off + (long long)(rr / BK) * IMG;
                const int rp = rr % BM, rq = rr % BK;
                for (int r = 0; r < nrhs; r++) {
                    const double *xr = x + r * rh.x_ld + row_off;
                    double *pp = bases.p[BASE_XP] + r * rh.stride[BASE_XP] + po, *pq = bases.p[BASE_XQ] + r * rh.stride[BASE_XQ] + qo;
                    constexpr int U = 8;
                    for (int c0 = lane; c0 < dk; c0 += 32 * U) {
                        double v[U];
#pragma unroll
                        for (int q = 0; q < U; q++) { const int c = c0 + 32 * q; v[q] = c < dk ? xr[c] : 0.0; }
#pragma unroll
                        for (int q = 0; q < U; q++) {
                            const int c = c0 + 32 * q;
                            if (c >= dk) break;
                            pp[(long long)(c / BK) * IMG + img_p_index(rp, c % BK)] = v[q];
                            pq[(long long)(c / BN) * KTq * IMG + img_q_index(rq, c % BN)] = v[q];
                        }
                    }
                }
            }
        } else
        for (int r = 0; r < nrhs; r++)
            ximg_share(segs, n_xsegs, x + r * rh.x_ld, lo, min(n, lo + share), bases.p[BASE_XP] + r * rh.stride[BASE_XP],
                       bases.p[BASE_XQ] + r * rh.stride[BASE_XQ], tid);
        fence_proxy_async();
        __threadfence();
        __syncthreads();
        if (tid == 0) atomicAdd(&ctrl[CTRL_XREADY], 1);
    } else {
        __syncthreads();       // the mbarrier initialisation above
    }
    if (xmode == 2 && (int)blockIdx.x < xs.n_loaders) {
        // Streamed input: x lives in pinned host memory.  A few loader CTAs (few, so that the shares arrive over PCIe in the order
        // they were requested) pull it share by share in the order of first use, write the tile images and the device copy,
        // and publish the elements written per 16-row block of every segment; the units' X items wait for exactly the row blocks they
        // read next (begin_item, wait_row_blocks).  A loader
        // waits for nothing, and joins the others on the units once the share list is empty.
        __shared__ int s_share;
        for (;;) {
            __syncthreads();
            if (tid == 0) s_share = atomicAdd(&ctrl[CTRL_XSHARE], 1);
            __syncthreads();
            const int sh = s_share;
            if (sh >= xs.n_shares) break;
            const XShare S = xs.shares[sh];
            const XSeg sg = xsegs[S.seg];
            const int KTp = (sg.dk + BK - 1) / BK, KTq = (sg.di + BK - 1) / BK;
            constexpr int U = 12;
            double v[U];
#pragma unroll
            for (int q = 0; q < U; q++) { const int e = S.lo + tid + q * THREADS; v[q] = e < S.hi ? x[sg.seg_off + e] : 0.0; }
#pragma unroll
            for (int q = 0; q < U; q++) {
                const int e = S.lo + tid + q * THREADS;
                if (e >= S.hi) break;
                const int r = e / sg.dk, c = e - r * sg.dk;
                bases.p[BASE_XP][sg.xp_off + ((long long)(r / BM) * KTp + c / BK) * IMG + img_p_index(r % BM, c % BK)] = v[q];
                bases.p[BASE_XQ][sg.xq_off + ((long long)(c / BN) * KTq + r / BK) * IMG + img_q_index(r % BK, c % BN)] = v[q];
                if (xs.x_copy) xs.x_copy[sg.seg_off + e] = v[q];
            }
            fence_proxy_async();
            __threadfence();
            __syncthreads();
            {   // elements of this share per row block of the segment
                const int b0 = (S.lo / sg.dk) / BK, b1 = ((S.hi - 1) / sg.dk) / BK;
                for (int b = b0 + tid; b <= b1; b += THREADS) {
                    const int lo_b = max(S.lo, b * BK * sg.dk), hi_b = min(S.hi, min((b + 1) * BK, sg.di) * sg.dk);
                    if (hi_b > lo_b) atomicAdd(&xs.xrb[sg.rb0 + b], hi_b - lo_b);
                }
            }
        }
    }
    if (ctr && tid == 0) ctr[1] = globaltimer();

    if (warp == CONSUMERS / 32) {
        // ================================================= producer
        if (lane == 0 && !skip_phase0) {
            long long spins = 0;
            while (ld_acquire(&ctrl[CTRL_XREADY]) < (int)gridDim.x) {
                __nanosleep(32);
                if (++spins > (1ll << 26)) { atomicExch(err, 1); break; }
            }
        }
        __syncwarp();
        fence_proxy_async();
        if (ctr && lane == 0) ctr[2] = globaltimer();
        int g = 0;                                   // stages issued so far
        auto acquire = [&]() {                       // waits until the consumers have released the stage; returns its index
            const int s = g % STAGES;
            if (g >= STAGES) mbar_wait(smem_u32(bars + STAGES + s), ((g / STAGES) & 1) ^ 1);
            return s;
        };
        for (;;) {
            int ticket = 0;
            if (lane == 0) ticket = atomicAdd(&ctrl[CTRL_TICKET], 1);
            ticket = __shfl_sync(0xffffffffu, ticket, 0);
            if (ticket >= n_units * nrhs) break;
            const int rhs = ticket % nrhs;               // ticket = unit * nrhs + rhs: a unit waits on smaller tickets only
            const int uw = lane < UNIT_WORDS ? reinterpret_cast<const int *>(units + ticket / nrhs)[lane] : 0;
#define UFIELD(f) __shfl_sync(0xffffffffu, uw, (int)(offsetof(GemmUnit, f) / 4))
            const int M = UFIELD(M), N = UFIELD(N), m0 = UFIELD(m0), n0 = UFIELD(n0);
            (void)0;
            const int item_begin = UFIELD(item_begin), item_count = UFIELD(item_count);
            const int KT = UFIELD(kt_count);
            int p_item = UFIELD(item0);
            const int k00 = UFIELD(k00);
            const int n_split = UFIELD(n_split), split_idx = UFIELD(split_idx), tile_id = UFIELD(tile_id);
            const int part_lo = UFIELD(part_off), part_hi = __shfl_sync(0xffffffffu, uw, (int)(offsetof(GemmUnit, part_off) / 4) + 1);
            const bool reducer = n_split > 1 && ((UFIELD(c_base) >> 24) & 1);     // GemmUnit::reducer is the 4th byte of that word
#undef UFIELD
            const int ext_m = min(BM, M - m0), ext_n = min(BN, N - n0);
            const int rot = ((m0 >> 6) + (n0 >> 6)) & (CWARPS - 1);     // the same for every K slice of a tile
            int layout = 0;                                             // 0: 4x2, 1: 2x4, 2: 8x1, 3: 1x8 sub-tiles per warp
            {
                const int sm = (ext_m + 7) >> 3, sn = (ext_n + 7) >> 3;
                int best = min(4, sm) * min(2, sn);
                if (min(2, sm) * min(4, sn) < best) { best = min(2, sm) * min(4, sn); layout = 1; }
                if (sm < best) { best = sm; layout = 2; }
                if (sn < best) { best = sn; layout = 3; }
            }
            const GemmItem *uitems = items + item_begin;
            if (KT == 0) {                           // an output without records: the consumers store zeros
                const int s = acquire();
                StageHdr *h = hdrs + s;
                if (lane == 0) { h->flags = F_FIRST | F_LAST; h->ticket = ticket; h->ext_m = ext_m; h->ext_n = ext_n; h->rot = rot; h->layout = layout; h->rhs = rhs; }
                if (lane < UNIT_WORDS) h->u[lane] = uw;
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(bars + s));
                g++;
                continue;
            }
            Producer pr{};
            begin_item(pr, uitems + p_item, s_base, s_stride, rhs, n_deps, m0, n0, k00, lane, ctrl, err, xmode, xsegs, xs.xrb);
            for (int t = 0; t < KT;) {
                // up to KPS consecutive k-tiles of the current item: their P images are contiguous, and so are their Q images
                // (a short group comes FIRST: the last stage of an item, and so of the unit, is a full one, which gives the
                // producer the longest possible cover for its trips to L2 at the boundary)
                const int rem = min((pr.K - pr.k0 + BK - 1) / BK, KT - t);
                const int nk = (rem % KPS) ? rem % KPS : KPS;
                if (pr.xq_dk > 0) wait_row_blocks(xs.xrb, pr.xq_rb0, pr.xq_di, pr.xq_dk, pr.k0 / BK, nk, lane, err);
                const int s = acquire();
                StageHdr *h = hdrs + s;
                const bool last = (t + nk == KT) && !reducer;
                if (lane == 0) { h->flags = F_DATA | (t == 0 ? F_FIRST : 0) | (last ? F_LAST : 0); h->ticket = ticket; h->ext_m = ext_m; h->ext_n = ext_n; h->rot = rot; h->layout = layout; h->rhs = rhs; h->nk = nk; }
                if (last && lane < UNIT_WORDS) h->u[lane] = uw;
                __syncwarp();
                if (lane == 0) {
                    const unsigned sP = smem_u32(stage_base + (size_t)s * STAGE_DOUBLES), bar = smem_u32(bars + s);
                    mbar_arrive_expect_tx(bar, (unsigned)nk * 2 * IMG * 8);
                    bulk_g2s(sP, pr.pP, (unsigned)nk * IMG * 8, bar);
                    bulk_g2s(sP + KPS * IMG * 8, pr.pQ, (unsigned)nk * IMG * 8, bar);
                }
                pr.pP += nk * IMG; pr.pQ += nk * IMG; pr.k0 += nk * BK;
                t += nk;
                g++;
                if (pr.k0 >= pr.K && t < KT) {
                    p_item++;
                    if (p_item < item_count) begin_item(pr, uitems + p_item, s_base, s_stride, rhs, n_deps, m0, n0, 0, lane, ctrl, err, xmode, xsegs, xs.xrb);
                }
            }
            if (reducer) {
                // split K, designated reducer (the slice of the tile that comes last in ticket order): once the other
                // n_split - 1 slices have parked their partial tiles (one arrival per consumer warp each), stream them
                // through the ring -- 32 KB per slice, one stage -- and let the consumers add them to their registers IN
                // SLICE ORDER (fixed at plan time: bitwise independent of timing, A22/A23).  The wait is on smaller tickets only.
                if (lane == 0) {
                    int *c = counters + rhs * rh.n_counters + tile_id;
                    const int need = CWARPS * (n_split - 1);
                    long long spins = 0;
                    while (ld_acquire(c) < need) {
                        __nanosleep(32);
                        if (++spins > (1ll << 26)) { atomicExch(err, 1); break; }
                    }
                    *c = 0;                          // self-cleaning for the next launch (this unit is the only reader)
                }
                __syncwarp();
                fence_proxy_async();
                const double *part = s_base[BASE_PART] + rhs * s_stride[BASE_PART] + (((long long)part_hi << 32) | (unsigned)part_lo);
                int r = 0;
                for (int sl = 0; sl < n_split; sl++) {
                    if (sl == split_idx) continue;
                    const int s = acquire();
                    StageHdr *h = hdrs + s;
                    const bool last = (++r == n_split - 1);
                    if (lane == 0) { h->flags = F_REDUCE | (last ? F_LAST : 0); h->ticket = ticket; h->ext_m = ext_m; h->ext_n = ext_n; h->rot = rot; h->layout = layout; h->rhs = rhs; h->nk = 0; }
                    if (last && lane < UNIT_WORDS) h->u[lane] = uw;
                    __syncwarp();
                    if (lane == 0) {
                        const unsigned bar = smem_u32(bars + s);
                        mbar_arrive_expect_tx(bar, BM * BN * 8);
                        bulk_g2s(smem_u32(stage_base + (size_t)s * STAGE_DOUBLES), part + (long long)sl * (BM * BN), BM * BN * 8, bar);
                    }
                    g++;
                }
            }
        }
        {   // no more tickets: tell the consumers to leave
            const int s = acquire();
            if (lane == 0) hdrs[s].flags = F_EXIT;
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(bars + s));
        }
        if (pf.base) {
            // side job while the launch drains (the ticket queue is empty, HBM is idle): L2 prefetch of this CTA's slice
            // of the rows the next kernel streams first; fire and forget, 128-byte lines
            const long long lines = (pf.rows + 15) >> 4;
            const long long l0 = lines * blockIdx.x / gridDim.x, l1 = lines * (blockIdx.x + 1) / gridDim.x;
            for (int c = 0; c < pf.cols; c++) {
                const double *col = pf.base + (long long)c * pf.ld;
                for (long long l = l0 + lane; l < l1; l += 32)
                    asm volatile("prefetch.global.L2 [%0];" ::"l"(col + (l << 4)));
            }
        }
    } else {
        // ================================================= consumers
        // Warp -> block of sub-tiles: w = (warp + rot) mod 8 in the warp grid of the unit's layout.  The rotation changes
        // from tile to tile so that the light warps of edge tiles do not always land on the same SM sub-partition (each
        // has its own DMMA pipe).
        const int gq = lane >> 2, tg = lane & 3;
        Lane L;
#pragma unroll
        for (int k4 = 0; k4 < 4; k4++) L.offA[k4] = gq * BK + ((((2 * k4 + (tg >> 1)) ^ (2 * (gq & 3)))) << 1) + (tg & 1);
        L.rowB = tg * BN + (gq & 1); L.c0 = gq >> 1; L.x2 = 2 * tg;

        double acc[8][2];
#pragma unroll
        for (int q = 0; q < 8; q++) { acc[q][0] = 0.0; acc[q][1] = 0.0; }
        unsigned long long t_start = 0, t_main = 0;

        // Deferred publish: a finished tile (a T-block tile, or a parked split-K partial) is announced by this WARP on its
        // own -- fence, then one atomic per warp; the counters count warps -- at the head of a later stage (PUBLISH_DELAY), or as
        // soon as the warp would block.
        int *pending = nullptr; int pending_g = 0;
        auto flush = [&]() {
            if (pending) {
                fence_proxy_async();      // readers pull these bytes with the TMA unit (async proxy)
                __threadfence();
                __syncwarp();
                if (lane == 0) atomicAdd(pending, 1);
                pending = nullptr;
            }
        };
        for (int g = 0;; g++) {
            const int s = g % STAGES;
            if (pending && (g - pending_g >= PUBLISH_DELAY || !mbar_test(smem_u32(bars + s), (g / STAGES) & 1))) flush();
            mbar_wait(smem_u32(bars + s), (g / STAGES) & 1);
            const StageHdr *h = hdrs + s;
            const int flags = h->flags;
            if (flags & F_EXIT) break;
            if (trace && tid == 0 && (flags & F_FIRST)) t_start = globaltimer();
            const int w = (warp + h->rot) & (CWARPS - 1);
            const int layout = h->layout;
            // first sub-tile row / column of this warp: 4x2 -> grid 2x4, 2x4 -> 4x2, 8x1 -> 1x8, 1x8 -> 8x1
            const int sr0 = layout == 0 ? (w & 1) * 4 : (layout == 1 ? (w & 3) * 2 : (layout == 2 ? 0 : w));
            const int sc0 = layout == 0 ? (w >> 1) * 2 : (layout == 1 ? (w >> 2) * 4 : (layout == 2 ? w : 0));
            if (flags & F_DATA) {
                // sub-tiles of this warp's block that hold real rows / columns: exactly those are multiplied
                const int mi = ((h->ext_m + 7) >> 3) - sr0, nj = ((h->ext_n + 7) >> 3) - sc0;
                if (mi > 0 && nj > 0) {
                    const int nk = h->nk;
                    const double *sP = stage_base + (size_t)s * STAGE_DOUBLES + sr0 * 8 * BK;
                    const double *sQ = stage_base + (size_t)s * STAGE_DOUBLES + KPS * IMG;
                    if (layout == 0 && mi >= 4 && nj >= 2 && nk == KPS) {
                        // the common case, a full stage of a full block: KPS k-tiles as one straight-line instruction stream
#pragma unroll
                        for (int kk = 0; kk < KPS; kk++) mma_ktile<4, 2, 2>(acc, sP + kk * IMG, sQ + kk * IMG, L, sc0);
                    } else {
#pragma unroll 1
                        for (int kk = 0; kk < nk; kk++, sP += IMG, sQ += IMG) {
                            if (layout == 0) disp_nj<4, 2, 2>(min(mi, 4), min(nj, 2), acc, sP, sQ, L, sc0);
                            else if (layout == 1) disp_nj<2, 4, 4>(min(mi, 2), min(nj, 4), acc, sP, sQ, L, sc0);
                            else if (layout == 2) disp_nj<8, 1, 1>(min(mi, 8), 1, acc, sP, sQ, L, sc0);
                            else disp_nj<1, 8, 8>(1, min(nj, 8), acc, sP, sQ, L, sc0);
                        }
                    }
                }
            } else if (flags & F_REDUCE) {
                // another slice's partial tile, in fragment order [register pair][thread]: add it in place
                const double2 *src = reinterpret_cast<const double2 *>(stage_base + (size_t)s * STAGE_DOUBLES) + tid;
#pragma unroll
                for (int q = 0; q < 8; q++) { const double2 v = src[q * CONSUMERS]; acc[q][0] += v.x; acc[q][1] += v.y; }
            }
            if (flags & F_LAST) {
                const GemmUnit &u = *reinterpret_cast<const GemmUnit *>(h->u);
                if (trace && tid == 0) t_main = globaltimer();
                flush();
                const bool writes_c = !(u.n_split > 1 && !u.reducer);
                if (!writes_c) {
                    // split K, not the reducer: park the partial tile (fragment order: [slice][register pair][thread], coalesced
                    // 16-byte stores) for the tile's designated reducer
                    double2 *mine = reinterpret_cast<double2 *>(s_base[BASE_PART] + h->rhs * s_stride[BASE_PART] + u.part_off) +
                                    (long long)u.split_idx * (BM * BN / 2);
#pragma unroll
                    for (int q = 0; q < 8; q++) __stcg(mine + q * CONSUMERS + tid, make_double2(acc[q][0], acc[q][1]));
                    pending = counters + h->rhs * rh.n_counters + u.tile_id; pending_g = g;
                } else {
                    double *C = s_base[u.c_base] + h->rhs * s_stride[u.c_base] + u.c_off;
                    const double *xr = x + h->rhs * rh.x_ld;
                    if (layout == 0) store_c<4, 2>(acc, u, C, sr0, sc0, gq, tg, yvec, axpy, xr);
                    else if (layout == 1) store_c<2, 4>(acc, u, C, sr0, sc0, gq, tg, yvec, axpy, xr);
                    else if (layout == 2) store_c<8, 1>(acc, u, C, sr0, sc0, gq, tg, yvec, axpy, xr);
                    else store_c<1, 8>(acc, u, C, sr0, sc0, gq, tg, yvec, axpy, xr);
                    // this tile of a T block is complete: to be published (release: this warp's stores, then its count)
                    if (u.signal >= 0) { pending = ctrl + CTRL_DEP0 + h->rhs * n_deps + u.signal; pending_g = g; }
                }
                if (trace && tid == 0) {
                    unsigned long long *tr = trace + 4ull * h->ticket;
                    tr[0] = t_start; tr[1] = t_main; tr[2] = globaltimer();
                    // bits 0-15 SM id, 16-31 k-tiles of the unit, 32-47 CTA, 48 stage-1 unit, 49 split-K unit, 50 wrote C
                    tr[3] = smid() | ((unsigned long long)u.kt_count << 16) | ((unsigned long long)blockIdx.x << 32) |
                            ((unsigned long long)(u.signal >= 0) << 48) | ((unsigned long long)(u.n_split > 1) << 49) |
                            ((unsigned long long)writes_c << 50) | ((unsigned long long)((h->ext_m + 7) >> 3) << 52) |
                            ((unsigned long long)((h->ext_n + 7) >> 3) << 56);      // bits 52-55 / 56-59: sub-tile rows / columns with data
                }
#pragma unroll
                for (int q = 0; q < 8; q++) { acc[q][0] = 0.0; acc[q][1] = 0.0; }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(bars + STAGES + s));     // this warp is done with the stage
        }
        flush();
    }
    // every unit this CTA took is finished; the last CTA to get here resets the control words for the next launch
    __syncthreads();
    if (ctr && tid == 0) ctr[3] = globaltimer();
    if (tid == 0) {
        __threadfence();
        const int fin = atomicAdd(&ctrl[CTRL_FINISHED], 1);
        s_is_last = (fin == (int)gridDim.x - 1);
    }
    __syncthreads();
    if (s_is_last) {
        for (int e = tid; e < CTRL_DEP0 + n_deps * nrhs; e += THREADS) ctrl[e] = 0;
        if (xmode == 2) for (int e = tid; e < xs.n_xrb; e += THREADS) xs.xrb[e] = 0;
    }
}

}  // namespace

// kernel variants (selected once per process; DMRG_GEMM_VARIANT overrides the default for experiments)
typedef void (*gemm_fn)(const GemmUnit *, const GemmItem *, BasePtrs, int *, int *, int, int, const int *, int,
                        unsigned long long *, Prefetch, int *, const XSeg *, int, const double *, long long, RhsInfo, int, const AxpyItem *,
                        XStream);
struct Variant { const char *name; gemm_fn fn; int smem; int ctas_per_sm; };
static const Variant kVariants[] = {
    {"s2b2", grouped_gemm_kernel<2, 2>, smem_bytes(2), 2},     // default: two CTAs per SM, two stages of three k-tiles (48 KB) each
    {"s3b1", grouped_gemm_kernel<3, 1>, smem_bytes(3), 1},
    {"s4b1", grouped_gemm_kernel<4, 1>, smem_bytes(4), 1},
};
static const Variant *g_variant = &kVariants[0];
static int g_ctas_per_sm = 0;

cudaError_t gemm_kernel_setup() {
    if (const char *e = getenv("DMRG_GEMM_VARIANT"))
        for (const Variant &v : kVariants)
            if (std::string(v.name) == e) g_variant = &v;
    for (const Variant &v : kVariants) {
        cudaError_t err = cudaFuncSetAttribute(v.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, v.smem);
        if (err != cudaSuccess) return err;
    }
    int occ = 0;
    cudaError_t err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, g_variant->fn, THREADS, g_variant->smem);
    if (err != cudaSuccess) return err;
    g_ctas_per_sm = std::max(1, std::min(occ, g_variant->ctas_per_sm));
    if (const char *e = getenv("DMRG_CTAS_PER_SM")) g_ctas_per_sm = std::max(1, std::min(g_ctas_per_sm, atoi(e)));
    return cudaSuccess;
}

int apply_H(Plan *p, const double *x, double *y, const int *done_flag, cudaStream_t st, const Prefetch *pf_in,
            int nrhs, long long ldx, long long ldy, bool trust_images) {
    // the tile images of x are current only if the library wrote them itself for exactly this vector (Plan::ximg_src)
    int xmode = (trust_images && nrhs == 1 && p->ximg_src == x) ? 1 : 0;
    p->ximg_src = nullptr;
    // dmrg_davidson_step_host: x is streamed from pinned host memory (and copied to `x`)
    XStream xs{};
    const double *x_src = x;
    if (p->x_stream && nrhs == 1 && p->n_xshares > 0) {
        static const int loaders = []() { const char *e = getenv("DMRG_XLOADERS"); return e ? atoi(e) : 24; }();
        xmode = 2; x_src = p->x_stream;
        xs.shares = p->xshares; xs.n_shares = p->n_xshares; xs.n_loaders = std::max(1, loaders); xs.x_copy = const_cast<double *>(x);
        xs.xrb = p->xrb; xs.n_xrb = p->n_xrb;
    }
    p->x_stream = nullptr;
    {
        static const int p0_rows = []() { const char *e = getenv("DMRG_P0_ROWS"); return e ? atoi(e) : 1; }();
        if (p0_rows) { xs.xrows = p->xrows; xs.n_xrows = p->n_xrows; }
    }
    if (nrhs < 1 || nrhs > p->max_rhs) return fail(p, DMRG_E_INVALID_ARG, "apply_H: more right-hand sides than options.max_rhs");
    BasePtrs b;
    b.p[BASE_XP] = p->ximg_p;
    b.p[BASE_XQ] = p->ximg_q;
    b.p[BASE_Y] = y;
    b.p[BASE_T] = p->tws;
    b.p[BASE_POOL] = p->pool;
    b.p[BASE_PART] = p->part;
    cudaEvent_t *ev = p->timing.enabled ? p->timing.ev : nullptr;
    if (ev) cudaEventRecord(ev[0], st);
    const int n_units = p->n_units1 + p->n_units2;
    p->launches += n_units > 0 ? 1 : 0;
    if (n_units > 0) {
        const int yvec = ((reinterpret_cast<uintptr_t>(y) & 15) == 0 && (nrhs == 1 || ldy % 2 == 0)) ? 1 : 0;
        RhsInfo rh{};
        rh.nrhs = nrhs; rh.n_deps = p->n_deps; rh.n_counters = p->n_counters; rh.x_ld = ldx;
        rh.stride[BASE_XP] = p->xp_elems; rh.stride[BASE_XQ] = p->xq_elems; rh.stride[BASE_T] = p->tws_elems;
        rh.stride[BASE_PART] = p->part_elems; rh.stride[BASE_Y] = ldy; rh.stride[BASE_POOL] = 0;
        Prefetch pf;
        if (pf_in && pf_in->base && pf_in->cols > 0 && pf_in->rows > 0) pf = *pf_in;
        const int grid = (int)std::min<long long>((long long)n_units * nrhs, (long long)g_ctas_per_sm * p->sm_count);   // persistent: one wave
        xs.n_loaders = std::min(xs.n_loaders, grid);
        g_variant->fn<<<grid, THREADS, g_variant->smem, st>>>(xmode == 2 ? p->units_stream : p->units, p->items, b, p->counters, p->ctrl, n_units,
                                                              p->n_deps, done_flag, yvec, p->trace, pf, &p->state->gemm_error,
                                                              p->xsegs, p->n_xsegs, x_src, p->n, rh, xmode, p->axpy, xs);
    }
    if (ev) { cudaEventRecord(ev[1], st); cudaEventRecord(ev[2], st); }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(p, DMRG_E_CUDA, std::string("apply_H launch: ") + cudaGetErrorString(e));
    return DMRG_OK;
}

}  // namespace dmrg
