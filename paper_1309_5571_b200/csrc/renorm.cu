// renorm.cu -- the steps either side of the Davidson hot path in one infinite-lattice DMRG iteration:
// PAPER.md:L100-110, Alg. 1 -- line 2 "form the superblock configuration" (block enlargement by one site, L112-120),
// line 5 "construct the density matrix for the given block from the lowest eigenstate", line 6 "compute the eigenvalues of
// the density matrix", line 7 "renormalize the basis of the block by keeping states with high eigenvalues" -- and the loop
// over them for the open spin-1/2 Heisenberg chain (Eq. 1-3), with line 3 done by dmrg_lowest_eigenpair.
// The paper gives no formulas for these lines; the textbook definitions are restated in oracle/renorm.py (O-REN), which
// the parity tests compare against step by step.  These steps run once per DMRG iteration (the Davidson loop runs a few
// hundred projections in between: "> 97 %" of the time), so the kernels here are plain FP64 FMA tiles.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <map>
#include <vector>
#include <time.h>
#include <cstdio>
#include "internal.h"

namespace dmrg {

namespace {

constexpr int RT = 32;      // tile edge of the plain GEMM-shaped kernels

// ---------------------------------------------------------------- line 5: rho_s = sum X X^T (left) / sum X^T X (right)
struct DenSeg { long long x_off; int di, dk; };           // one segment X_ik (row-major d_i x d_k) of the target-sector vector
struct DenJob { long long rho_off; int d, seg_begin, seg_count; };   // one sector of the chosen side
__global__ void __launch_bounds__(RT * RT / 4)
density_kernel(const DenJob *__restrict__ jobs, const DenSeg *__restrict__ segs, const double *__restrict__ x, int side,
               double *__restrict__ rho) {
    const DenJob jb = jobs[blockIdx.z];
    const int a0 = blockIdx.y * RT, b0 = blockIdx.x * RT;
    if (a0 >= jb.d || b0 >= jb.d) return;
    __shared__ double sA[RT][RT + 1], sB[RT][RT + 1];     // [contraction index][a or b]
    const int tx = threadIdx.x % 16, ty = threadIdx.x / 16;   // 16 x 16 threads, 2 x 2 outputs each
    double acc[2][2] = {{0.0, 0.0}, {0.0, 0.0}};
    for (int s = 0; s < jb.seg_count; s++) {
        const DenSeg sg = segs[jb.seg_begin + s];
        const double *X = x + sg.x_off;
        const int K = side == 0 ? sg.dk : sg.di;          // contraction length: the OTHER side's dimension
        for (int k0 = 0; k0 < K; k0 += RT) {
            for (int e = threadIdx.x; e < RT * RT; e += RT * RT / 4) {
                const int kk = e / RT, c = e % RT;        // element (k0 + kk) of the contraction, row/col c of the tile
                double va = 0.0, vb = 0.0;
                if (k0 + kk < K) {
                    if (side == 0) {                      // left: rho[a][b] += X[a][k] X[b][k]
                        if (a0 + c < jb.d) va = X[(long long)(a0 + c) * sg.dk + k0 + kk];
                        if (b0 + c < jb.d) vb = X[(long long)(b0 + c) * sg.dk + k0 + kk];
                    } else {                              // right: rho[a][b] += X[k][a] X[k][b]
                        if (a0 + c < jb.d) va = X[(long long)(k0 + kk) * sg.dk + a0 + c];
                        if (b0 + c < jb.d) vb = X[(long long)(k0 + kk) * sg.dk + b0 + c];
                    }
                }
                sA[kk][c] = va; sB[kk][c] = vb;
            }
            __syncthreads();
#pragma unroll 8
            for (int kk = 0; kk < RT; kk++) {
                const double a_0 = sA[kk][2 * ty], a_1 = sA[kk][2 * ty + 1], b_0 = sB[kk][2 * tx], b_1 = sB[kk][2 * tx + 1];
                acc[0][0] = fma(a_0, b_0, acc[0][0]); acc[0][1] = fma(a_0, b_1, acc[0][1]);
                acc[1][0] = fma(a_1, b_0, acc[1][0]); acc[1][1] = fma(a_1, b_1, acc[1][1]);
            }
            __syncthreads();
        }
    }
    double *R = rho + jb.rho_off;
    for (int i = 0; i < 2; i++) for (int j = 0; j < 2; j++) {
        const int a = a0 + 2 * ty + i, b = b0 + 2 * tx + j;
        if (a < jb.d && b < jb.d) R[(long long)a * jb.d + b] = acc[i][j];
    }
}

// ---------------------------------------------------------------- line 7: batched C = op(A) B (plain tiles, one job per z)
struct MmJob { const double *A, *B; double *C; int lda, ldb, ldc, M, N, K, transA; };
__global__ void __launch_bounds__(RT * RT / 4)
mm_kernel(const MmJob *__restrict__ jobs) {
    const MmJob jb = jobs[blockIdx.z];
    const int m0 = blockIdx.y * RT, n0 = blockIdx.x * RT;
    if (m0 >= jb.M || n0 >= jb.N) return;
    __shared__ double sA[RT][RT + 1], sB[RT][RT + 1];     // sA[k][m], sB[k][n]
    const int tx = threadIdx.x % 16, ty = threadIdx.x / 16;
    double acc[2][2] = {{0.0, 0.0}, {0.0, 0.0}};
    for (int k0 = 0; k0 < jb.K; k0 += RT) {
        for (int e = threadIdx.x; e < RT * RT; e += RT * RT / 4) {
            const int kk = e / RT, c = e % RT;
            double va = 0.0, vb = 0.0;
            if (k0 + kk < jb.K) {
                if (m0 + c < jb.M) va = jb.transA ? jb.A[(long long)(k0 + kk) * jb.lda + m0 + c] : jb.A[(long long)(m0 + c) * jb.lda + k0 + kk];
                if (n0 + c < jb.N) vb = jb.B[(long long)(k0 + kk) * jb.ldb + n0 + c];
            }
            sA[kk][c] = va; sB[kk][c] = vb;
        }
        __syncthreads();
#pragma unroll 8
        for (int kk = 0; kk < RT; kk++) {
            const double a_0 = sA[kk][2 * ty], a_1 = sA[kk][2 * ty + 1], b_0 = sB[kk][2 * tx], b_1 = sB[kk][2 * tx + 1];
            acc[0][0] = fma(a_0, b_0, acc[0][0]); acc[0][1] = fma(a_0, b_1, acc[0][1]);
            acc[1][0] = fma(a_1, b_0, acc[1][0]); acc[1][1] = fma(a_1, b_1, acc[1][1]);
        }
        __syncthreads();
    }
    for (int i = 0; i < 2; i++) for (int j = 0; j < 2; j++) {
        const int m = m0 + 2 * ty + i, n = n0 + 2 * tx + j;
        if (m < jb.M && n < jb.N) jb.C[(long long)m * jb.ldc + n] = acc[i][j];
    }
}

// ---------------------------------------------------------------- line 2: scaled placement of blocks (enlargement)
// dst[r0 + i][c0 + j] += scale * src[i][j] (or src[j][i]); src == nullptr places scale * identity (rows x rows)
struct PlaceJob { const double *src; double *dst; int lds, ldd, rows, cols, r0, c0, transpose; double scale; };
__global__ void place_kernel(const PlaceJob *__restrict__ jobs) {
    const PlaceJob jb = jobs[blockIdx.y];
    const long long tot = jb.src ? (long long)jb.rows * jb.cols : jb.rows;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < tot; e += (long long)gridDim.x * blockDim.x) {
        if (!jb.src) { jb.dst[(long long)(jb.r0 + e) * jb.ldd + jb.c0 + e] += jb.scale; continue; }
        const int i = (int)(e / jb.cols), j = (int)(e % jb.cols);
        const double v = jb.transpose ? jb.src[(long long)j * jb.lds + i] : jb.src[(long long)i * jb.lds + j];
        jb.dst[(long long)(jb.r0 + i) * jb.ldd + jb.c0 + j] += jb.scale * v;
    }
}

// ---------------------------------------------------------------- line 6: all eigenpairs of every sector block
// Cyclic Jacobi with the round-robin (parallel) ordering, one CTA per sector, the matrix in global memory (L2): per round
// d/2 disjoint rotations J, applied as A <- A J (column phase: pair x row), then A <- J^T A (row phase: pair x column),
// E <- E J.  Converged when off(A)^2 <= (d eps)^2 ||A||_F^2.  Output: eigenvalues DESCENDING (ties: lower original column
// first) and the eigenvectors as columns of U in that order.  (The paper's own code uses Lanczos here; any symmetric
// eigensolver returns the same pairs.  This one is written for correctness: it runs once per DMRG iteration.)
struct EigJob { long long off; long long w_off; int d; };      // A, E, U at `off` (d x d row-major), w at w_off
constexpr int ET = 1024;
__device__ __forceinline__ void rot_pair(double app, double aqq, double apq, double &c, double &s) {
    c = 1.0; s = 0.0;
    if (apq == 0.0) return;
    const double tau = (aqq - app) / (2.0 * apq);
    if (!(fabs(tau) < 1e300)) return;
    const double t = copysign(1.0, tau) / (fabs(tau) + sqrt(fma(tau, tau, 1.0)));
    c = 1.0 / sqrt(fma(t, t, 1.0)); s = t * c;
}
__global__ void __launch_bounds__(ET)
sector_eig_kernel(const EigJob *__restrict__ jobs, double *__restrict__ Aall, double *__restrict__ Eall, double *__restrict__ Uall,
                  double *__restrict__ wall, int *__restrict__ status, int hdr_half, long long mat_doubles) {
    extern __shared__ unsigned char eig_smem[];
    const EigJob jb = jobs[blockIdx.x];
    const int d = jb.d, tid = threadIdx.x;
    if (d == 0) return;
    double *A = Aall + jb.off, *E = Eall + jb.off, *U = Uall + jb.off, *w = wall + jb.w_off;
    const int n = (d + 1) & ~1, half = n / 2;
    double *s_c = reinterpret_cast<double *>(eig_smem);          // [hdr_half]
    double *s_s = s_c + hdr_half;                                // [hdr_half]
    int *s_p = reinterpret_cast<int *>(s_s + hdr_half);          // [hdr_half]
    int *s_q = s_p + hdr_half;                                   // [hdr_half]
    __shared__ double s_red[2][ET / 32];
    __shared__ int s_stop;
    // The sweeps read and write every element of A and E 3 (n - 1) times with a CTA barrier in between: out of global memory a
    // round is three L2 round trips (~9 us at d = 190).  When they fit, A -- and E too -- live in shared memory for the whole
    // solve (mat_doubles doubles were allocated behind the header): d <= 118 both, d <= 167 A alone.
    {
        double *mat = reinterpret_cast<double *>(s_q + hdr_half);      // 24 hdr_half bytes in: 8-byte aligned
        const long long dd = (long long)d * d;
        if (dd <= mat_doubles) {
            for (long long e = tid; e < dd; e += ET) mat[e] = A[e];
            A = mat;
            if (2 * dd <= mat_doubles) E = mat + dd;
        }
    }
    for (long long e = tid; e < (long long)d * d; e += ET) E[e] = (e / d == e % d) ? 1.0 : 0.0;
    __syncthreads();
    int sweep = 0;
    for (; sweep < 60; sweep++) {
        double off = 0.0, dg = 0.0;
        for (long long e = tid; e < (long long)d * d; e += ET) { const double v = A[e]; if (e / d == e % d) dg = fma(v, v, dg); else off = fma(v, v, off); }
        for (int o = 16; o > 0; o >>= 1) { off += __shfl_xor_sync(0xffffffffu, off, o); dg += __shfl_xor_sync(0xffffffffu, dg, o); }
        if ((tid & 31) == 0) { s_red[0][tid >> 5] = off; s_red[1][tid >> 5] = dg; }
        __syncthreads();
        if (tid == 0) {
            double so = 0.0, sd = 0.0;
            for (int q = 0; q < ET / 32; q++) { so += s_red[0][q]; sd += s_red[1][q]; }
            s_stop = (so <= (double)d * d * 4.9e-32 * (so + sd)) ? 1 : 0;
        }
        __syncthreads();
        if (s_stop) break;
        for (int round = 0; round < n - 1; round++) {
            for (int t = tid; t < half; t += ET) {
                int p, q;
                if (t == 0) { p = n - 1; q = round; }
                else { p = (round + t) % (n - 1); q = (round - t + (n - 1)) % (n - 1); }
                if (p > q) { const int u = p; p = q; q = u; }
                double c = 1.0, s = 0.0;
                if (q < d) rot_pair(A[(long long)p * d + p], A[(long long)q * d + q], A[(long long)p * d + q], c, s);
                s_p[t] = p; s_q[t] = q; s_c[t] = c; s_s[t] = s;
            }
            __syncthreads();
            // One phase for A' = J^T A J: the rotations of a round act on disjoint index pairs, so A splits into half x half blocks
            // of 2 x 2 elements (rows of pair t1, columns of pair t2) that are updated independently and in place: columns first,
            // (x_P, x_Q) <- (c2 x_P - s2 x_Q, s2 x_P + c2 x_Q), then rows, (y_p, y_q) <- (c1 y_p - s1 y_q, s1 y_p + c1 y_q).
            for (long long e = tid; e < (long long)half * half; e += ET) {
                const int t1 = (int)(e / half), t2 = (int)(e % half);
                const double c1 = s_c[t1], s1 = s_s[t1], c2 = s_c[t2], s2 = s_s[t2];
                if (s1 == 0.0 && s2 == 0.0) continue;
                const int p = s_p[t1], q = s_q[t1], P = s_p[t2], Q = s_q[t2];
                const bool hq = q < d, hQ = Q < d;           // (the partner of the odd one out does not exist)
                double *rp = A + (long long)p * d, *rq = A + (long long)q * d;
                double apP = rp[P], apQ = hQ ? rp[Q] : 0.0, aqP = hq ? rq[P] : 0.0, aqQ = (hq && hQ) ? rq[Q] : 0.0;
                const double bpP = c2 * apP - s2 * apQ, bpQ = s2 * apP + c2 * apQ;
                const double bqP = c2 * aqP - s2 * aqQ, bqQ = s2 * aqP + c2 * aqQ;
                rp[P] = c1 * bpP - s1 * bqP;
                if (hQ) rp[Q] = c1 * bpQ - s1 * bqQ;
                if (hq) { rq[P] = s1 * bpP + c1 * bqP; if (hQ) rq[Q] = s1 * bpQ + c1 * bqQ; }
            }
            // E' = E J (columns only), in the same phase
            for (long long e = tid; e < (long long)half * d; e += ET) {
                const int t = (int)(e % half), i = (int)(e / half);
                const int p = s_p[t], q = s_q[t];
                if (q >= d) continue;
                const double c = s_c[t], s = s_s[t];
                if (s == 0.0) continue;
                double *re = E + (long long)i * d; const double ep = re[p], eq = re[q];
                re[p] = c * ep - s * eq; re[q] = s * ep + c * eq;
            }
            __syncthreads();
        }
    }
    if (tid == 0 && sweep >= 60) atomicExch(status, 1);
    // eigenvalues descending, ties by original column; U(:, rank) = E(:, column)
    for (int col = tid; col < d; col += ET) {
        const double v = A[(long long)col * d + col];
        int rank = 0;
        for (int o = 0; o < d; o++) { const double u = A[(long long)o * d + o]; if (u > v || (u == v && o < col)) rank++; }
        w[rank] = v;
        for (int i = 0; i < d; i++) U[(long long)i * d + rank] = E[(long long)i * d + col];
    }
}

// ---------------------------------------------------------------- host side
#define RN_TRY(x) do { cudaError_t e__ = (x); if (e__ != cudaSuccess) return fail(nullptr, (e__ == cudaErrorMemoryAllocation) ? DMRG_E_ALLOC : DMRG_E_CUDA, \
    std::string(#x) + ": " + cudaGetErrorString(e__)); } while (0)

template <class T> struct DevBuf {          // device array that lives as long as the object
    T *p = nullptr; size_t n = 0;
    DevBuf() {}
    DevBuf(const DevBuf &) = delete; DevBuf &operator=(const DevBuf &) = delete;
    ~DevBuf() { cudaFree(p); }
    cudaError_t alloc(size_t count, bool zero = false) {
        cudaFree(p); p = nullptr; n = count;
        cudaError_t e = cudaMalloc((void **)&p, std::max<size_t>(count, 1) * sizeof(T));
        if (e == cudaSuccess && zero) e = cudaMemset(p, 0, std::max<size_t>(count, 1) * sizeof(T));
        return e;
    }
    cudaError_t upload(const std::vector<T> &v, cudaStream_t st) {
        cudaError_t e = alloc(v.size());
        if (e == cudaSuccess && !v.empty()) e = cudaMemcpyAsync(p, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);      // v may be a temporary of the caller
        return e;
    }
};

}  // namespace

// rho of one side of the plan's superblock from the target-sector vector x (layout of dmrg_get_layout): sector s of that side
// at rho + rho_off[s], row-major d_s x d_s (zero matrix when the sector takes part in no pair).
int density_matrix(Plan *p, const double *x, int side, double *rho, cudaStream_t st) {
    const std::vector<int> &dims = side == 0 ? p->dimL : p->dimR;
    const int ns = (int)dims.size();
    std::vector<DenJob> jobs(ns); std::vector<DenSeg> segs;
    long long off = 0; int dmax = 1;
    for (int s = 0; s < ns; s++) {
        jobs[s] = {off, dims[s], (int)segs.size(), 0};
        for (size_t q = 0; q < p->pairL.size(); q++)
            if ((side == 0 ? p->pairL[q] : p->pairR[q]) == s) { segs.push_back({p->segOff[q], p->dimL[p->pairL[q]], p->dimR[p->pairR[q]]}); jobs[s].seg_count++; }
        off += (long long)dims[s] * dims[s]; dmax = std::max(dmax, dims[s]);
    }
    DevBuf<DenJob> dj; DevBuf<DenSeg> ds;
    RN_TRY(dj.upload(jobs, st)); RN_TRY(ds.upload(segs, st));
    const int tiles = (dmax + RT - 1) / RT;
    if (ns > 0) density_kernel<<<dim3(tiles, tiles, ns), RT * RT / 4, 0, st>>>(dj.p, ds.p, x, side, rho);
    RN_TRY(cudaGetLastError());
    RN_TRY(cudaStreamSynchronize(st));       // the job tables go out of scope
    return DMRG_OK;
}

// All eigenpairs of n_sectors symmetric blocks (concatenated d_s x d_s row-major, destroyed): U (same layout, columns by
// descending eigenvalue), w (concatenated, descending per sector).
int sector_eig(int ns, const int *dims, double *rho, double *U, double *w, cudaStream_t st) {
    std::vector<EigJob> jobs(ns);
    long long off = 0, woff = 0; int dmax = 1;
    for (int s = 0; s < ns; s++) { jobs[s] = {off, woff, dims[s]}; off += (long long)dims[s] * dims[s]; woff += dims[s]; dmax = std::max(dmax, dims[s]); }
    DevBuf<EigJob> dj; DevBuf<double> E; DevBuf<int> status;
    RN_TRY(dj.upload(jobs, st)); RN_TRY(E.alloc((size_t)off)); RN_TRY(status.alloc(1, true));
    const int half = ((dmax + 1) & ~1) / 2;
    const size_t hdr = (size_t)(half + (half & 1)) * (2 * sizeof(double) + 2 * sizeof(int));
    if (hdr > 200 * 1024) return fail(nullptr, DMRG_E_INVALID_ARG, "sector_eig: a sector larger than 12800 states");
    // shared memory behind the header for the matrices of the largest sector (both if they fit, else A alone, else none)
    const size_t cap = (size_t)225 * 1024 - hdr;
    const size_t dd = (size_t)dmax * dmax * sizeof(double);
    const size_t mat_bytes = 2 * dd <= cap ? 2 * dd : (dd <= cap ? dd : 0);
    const size_t smem = hdr + mat_bytes;
    RN_TRY(cudaFuncSetAttribute(sector_eig_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)std::max<size_t>(smem, 1024)));
    if (ns > 0) sector_eig_kernel<<<ns, ET, smem, st>>>(dj.p, rho, E.p, U, w, status.p, half, (long long)(mat_bytes / sizeof(double)));
    RN_TRY(cudaGetLastError());
    int hs = 0;
    RN_TRY(cudaMemcpyAsync(&hs, status.p, sizeof(int), cudaMemcpyDeviceToHost, st));
    RN_TRY(cudaStreamSynchronize(st));
    if (hs) return fail(nullptr, DMRG_E_NUMERIC, "sector_eig: Jacobi sweeps did not converge");
    return DMRG_OK;
}

// Alg. 1 line 7, the choice: the m largest eigenvalues over all sectors (reading A33: ties by sector index, then by rank inside
// the sector; eigenvalues <= 0 are never kept).  w: HOST, concatenated, descending per sector.
void select_states(int ns, const int *dims, const double *w, int m, int *m_keep, double *discarded) {
    struct C { double w; int s, r; };
    std::vector<C> c; double total = 0.0;
    long long off = 0;
    for (int s = 0; s < ns; s++) { for (int r = 0; r < dims[s]; r++) { total += w[off + r]; if (w[off + r] > 0.0) c.push_back({w[off + r], s, r}); } off += dims[s]; }
    std::stable_sort(c.begin(), c.end(), [](const C &a, const C &b) { if (a.w != b.w) return a.w > b.w; if (a.s != b.s) return a.s < b.s; return a.r < b.r; });
    for (int s = 0; s < ns; s++) m_keep[s] = 0;
    double kept = 0.0;
    for (size_t q = 0; q < c.size() && (int)q < m; q++) { m_keep[c[q].s]++; kept += c[q].w; }   // ranks are contiguous: w is descending per sector
    if (discarded) *discarded = total - kept;
}

// O'_b = U_dst(:, 0:m_dst)^T A_b U_src(:, 0:m_src) for every block of one operator (index arrays HOST, data DEVICE).
// out_data: DEVICE, the rotated blocks back to back (row-major m_dst x m_src, ld = m_src); out_offset HOST [n_blocks] (-1 for a
// block that disappears because one of its sectors keeps no state).  Returns the number of output elements in *out_elems.
int rotate_op(int ns, const int *dims, const int *m_keep, const double *U, int n_blocks, const int *src, const int *dst,
              const long long *offset, const int *ld, const double *data, double *out_data, long long *out_offset,
              long long *out_elems, cudaStream_t st) {
    std::vector<long long> uoff(ns + 1, 0);
    for (int s = 0; s < ns; s++) uoff[s + 1] = uoff[s] + (long long)dims[s] * dims[s];
    std::vector<MmJob> j1, j2; long long toff = 0, ooff = 0; int mmax = 1, nmax = 1, m2 = 1;
    for (int b = 0; b < n_blocks; b++) {
        const int s = src[b], d = dst[b];
        if (m_keep[s] == 0 || m_keep[d] == 0) { if (out_offset) out_offset[b] = -1; continue; }
        if (out_offset) out_offset[b] = ooff;
        // T (d_d x m_s) = A (d_d x d_s) U_s(:, 0:m_s);  out (m_d x m_s) = U_d(:, 0:m_d)^T T
        j1.push_back({data + offset[b], U + uoff[s], nullptr, ld[b], dims[s], m_keep[s], dims[d], m_keep[s], dims[s], 0});
        j2.push_back({U + uoff[d], nullptr, out_data ? out_data + ooff : nullptr, dims[d], m_keep[s], m_keep[s], m_keep[d], m_keep[s], dims[d], 1});
        j1.back().ldc = m_keep[s];
        j1.back().C = reinterpret_cast<double *>(toff);     // patched below once the scratch exists
        toff += (long long)dims[d] * m_keep[s]; ooff += (long long)m_keep[d] * m_keep[s];
        mmax = std::max(mmax, dims[d]); nmax = std::max(nmax, m_keep[s]); m2 = std::max(m2, m_keep[d]);
    }
    if (out_elems) *out_elems = ooff;
    if (!out_data || j1.empty()) return DMRG_OK;
    DevBuf<double> T; RN_TRY(T.alloc((size_t)toff));
    for (size_t q = 0; q < j1.size(); q++) { j1[q].C = T.p + reinterpret_cast<long long>(j1[q].C); j2[q].B = j1[q].C; }
    DevBuf<MmJob> d1, d2; RN_TRY(d1.upload(j1, st)); RN_TRY(d2.upload(j2, st));
    mm_kernel<<<dim3((nmax + RT - 1) / RT, (mmax + RT - 1) / RT, (unsigned)j1.size()), RT * RT / 4, 0, st>>>(d1.p);
    mm_kernel<<<dim3((nmax + RT - 1) / RT, (m2 + RT - 1) / RT, (unsigned)j2.size()), RT * RT / 4, 0, st>>>(d2.p);
    RN_TRY(cudaGetLastError());
    RN_TRY(cudaStreamSynchronize(st));
    return DMRG_OK;
}

// ---------------------------------------------------------------- blocks of the chain on the device, enlargement (line 2)
namespace {

struct DevOp {                     // sector-blocked operator: index arrays on the host, blocks back to back on the device
    std::vector<int> src, dst, ld; std::vector<long long> off; DevBuf<double> data; long long elems = 0;
    int add(int s, int d, int rows, int cols) { src.push_back(s); dst.push_back(d); ld.push_back(cols); off.push_back(elems); elems += (long long)rows * cols; return (int)src.size() - 1; }
    dmrg_block_op view() const { dmrg_block_op o; o.n_blocks = (int)src.size(); o.src = src.data(); o.dst = dst.data(); o.offset = reinterpret_cast<const int64_t *>(off.data()); o.ld = ld.data(); o.data = data.p; return o; }
};
struct DevBlock { std::vector<int> labels, dims; DevOp H, Sz, Sp; int n_sites = 0; };   // labels: 2 S_z

int run_places(std::vector<std::vector<PlaceJob>> &layers, cudaStream_t st) {
    for (auto &L : layers) {       // jobs of one layer write disjoint elements; layers accumulate in order
        if (L.empty()) continue;
        DevBuf<PlaceJob> dj; RN_TRY(dj.upload(L, st));
        place_kernel<<<dim3(8, (unsigned)L.size()), 256, 0, st>>>(dj.p);
        RN_TRY(cudaGetLastError()); RN_TRY(cudaStreamSynchronize(st));
    }
    return DMRG_OK;
}

int single_site(DevBlock &b, cudaStream_t st) {
    b.labels = {-1, 1}; b.dims = {1, 1}; b.n_sites = 1;
    b.Sz.add(0, 0, 1, 1); b.Sz.add(1, 1, 1, 1); b.Sp.add(0, 1, 1, 1);
    RN_TRY(b.H.data.alloc(0)); RN_TRY(b.Sz.data.upload({-0.5, 0.5}, st)); RN_TRY(b.Sp.data.upload({1.0}, st));
    return DMRG_OK;
}

// Enlarged block = block (x) site (left, block index slow) or site (x) block (right, site index slow), basis sorted by the label
// 2 S_z (stable in the composite index): new sector q' = [ (q'-1, up) ; (q'+1, down) ] on the left and [ (down, q'+1) ; (up, q'-1) ]
// on the right.  H_e = H_b + J/2 (S+_b S-_s + S-_b S+_s) + J Delta Sz_b Sz_s; the new site is the boundary site.
int enlarge(const DevBlock &b, int side, double J, double Delta, DevBlock &e, cudaStream_t st) {
    std::map<int, int> old_of;     // label -> old sector with d > 0
    for (size_t s = 0; s < b.labels.size(); s++) if (b.dims[s] > 0) old_of[b.labels[s]] = (int)s;
    std::map<int, int> new_of;
    for (auto &kv : old_of) { new_of[kv.first - 1] = 0; new_of[kv.first + 1] = 0; }
    e.labels.clear(); e.dims.clear(); e.n_sites = b.n_sites + 1;
    for (auto &kv : new_of) { kv.second = (int)e.labels.size(); e.labels.push_back(kv.first); e.dims.push_back(0); }
    auto dim_old = [&](int q) { auto it = old_of.find(q); return it == old_of.end() ? 0 : b.dims[it->second]; };
    // row offset of part (old label q, site spin sigma) inside new sector q + sigma
    auto part_off = [&](int q, int sigma) {
        if (side == 0) return sigma == +1 ? 0 : dim_old(q - 2);      // [ (q'-1, up) ; (q'+1, down) ]: down part follows the up part of label q-2
        return sigma == -1 ? 0 : dim_old(q + 2);                     // [ (down, q'+1) ; (up, q'-1) ]: up part follows the down part of label q+2
    };
    for (size_t n = 0; n < e.labels.size(); n++) e.dims[n] = dim_old(e.labels[n] - 1) + dim_old(e.labels[n] + 1);
    // allocate: H_e, Sz_e diagonal in the new sectors; Sp_e maps q' -> q' + 2
    std::vector<int> hblk(e.labels.size()), zblk(e.labels.size());
    for (size_t n = 0; n < e.labels.size(); n++) { hblk[n] = e.H.add((int)n, (int)n, e.dims[n], e.dims[n]); zblk[n] = e.Sz.add((int)n, (int)n, e.dims[n], e.dims[n]); }
    std::map<int, int> pblk;
    for (size_t n = 0; n < e.labels.size(); n++) { auto it = new_of.find(e.labels[n] + 2); if (it != new_of.end() && dim_old(e.labels[n] + 1) > 0) pblk[(int)n] = e.Sp.add((int)n, it->second, e.dims[it->second], e.dims[n]); }
    RN_TRY(e.H.data.alloc((size_t)e.H.elems, true)); RN_TRY(e.Sz.data.alloc((size_t)e.Sz.elems, true)); RN_TRY(e.Sp.data.alloc((size_t)e.Sp.elems, true));
    std::vector<std::vector<PlaceJob>> layers(3);
    auto Hdst = [&](int n) { return e.H.data.p + e.H.off[hblk[n]]; };
    // H_b and J Delta sigma/2 Sz_b on the diagonal parts
    for (size_t q = 0; q < b.H.src.size(); q++) {
        const int lab = b.labels[b.H.src[q]], d = b.dims[b.H.src[q]];
        for (int sg : {+1, -1}) { const int n = new_of[lab + sg], o = part_off(lab, sg); layers[0].push_back({b.H.data.p + b.H.off[q], Hdst(n), b.H.ld[q], e.dims[n], d, d, o, o, 0, 1.0}); }
    }
    for (size_t q = 0; q < b.Sz.src.size(); q++) {
        const int lab = b.labels[b.Sz.src[q]], d = b.dims[b.Sz.src[q]];
        for (int sg : {+1, -1}) { const int n = new_of[lab + sg], o = part_off(lab, sg); layers[1].push_back({b.Sz.data.p + b.Sz.off[q], Hdst(n), b.Sz.ld[q], e.dims[n], d, d, o, o, 0, J * Delta * 0.5 * sg}); }
    }
    // J/2 S+_b (q -> q+2) (x) S-_s: (q, up) -> (q+2, down) inside new sector q+1, and the transpose
    for (size_t q = 0; q < b.Sp.src.size(); q++) {
        const int ls = b.labels[b.Sp.src[q]], ldst = b.labels[b.Sp.dst[q]], ds = b.dims[b.Sp.src[q]], dd = b.dims[b.Sp.dst[q]];
        if (ds == 0 || dd == 0) continue;
        const int n = new_of[ls + 1], r0 = part_off(ldst, -1), c0 = part_off(ls, +1);
        layers[2].push_back({b.Sp.data.p + b.Sp.off[q], Hdst(n), b.Sp.ld[q], e.dims[n], dd, ds, r0, c0, 0, 0.5 * J});
        layers[2].push_back({b.Sp.data.p + b.Sp.off[q], Hdst(n), b.Sp.ld[q], e.dims[n], ds, dd, c0, r0, 1, 0.5 * J});
    }
    // Sz_e = 1 (x) Sz_s, Sp_e = 1 (x) S+_s: scaled identities on the parts
    for (auto &kv : old_of) {
        const int lab = kv.first, d = b.dims[kv.second];
        for (int sg : {+1, -1}) { const int n = new_of[lab + sg], o = part_off(lab, sg); layers[0].push_back({nullptr, e.Sz.data.p + e.Sz.off[zblk[n]], 0, e.dims[n], d, d, o, o, 0, 0.5 * sg}); }
        const int nsrc = new_of[lab - 1];           // (lab, down) in sector lab-1  ->  (lab, up) in sector lab+1
        auto it = pblk.find(nsrc);
        if (it != pblk.end()) layers[0].push_back({nullptr, e.Sp.data.p + e.Sp.off[it->second], 0, e.dims[nsrc], d, d, part_off(lab, +1), part_off(lab, -1), 0, 1.0});
    }
    return run_places(layers, st);
}

}  // namespace

// ---------------------------------------------------------------- Alg. 1 looped: infinite-lattice DMRG, Heisenberg chain
namespace {

static double g_t[8];
static double rn_now() { timespec ts; clock_gettime(CLOCK_MONOTONIC, &ts); return ts.tv_sec * 1e3 + ts.tv_nsec * 1e-6; }
#define RNT(i, st_) do { if (g_tdbg) { cudaStreamSynchronize(st_); double t_ = rn_now(); g_t[i] += t_ - g_tl; g_tl = t_; } } while (0)
static bool g_tdbg = false; static double g_tl = 0;
// Alg. 1 lines 4-7 for BOTH blocks of the superblock: the density matrices of the two sides, then ONE eigen-solver launch over
// the sectors of both (the launch lasts as long as its largest sector: two launches would take twice as long), then the choice of
// states and the rotations side by side.
int renormalise_both(Plan *p, const DevBlock &bl, const DevBlock &br, const double *x, int m, DevBlock &outl, DevBlock &outr,
                     double *disc_l, double *disc_r, cudaStream_t st) {
    const DevBlock *bs[2] = {&bl, &br};
    DevBlock *outs[2] = {&outl, &outr};
    double *disc[2] = {disc_l, disc_r};
    long long tot[2] = {0, 0}, wtot[2] = {0, 0};
    std::vector<int> dims_all;
    for (int side = 0; side < 2; side++)
        for (int d : bs[side]->dims) { tot[side] += (long long)d * d; wtot[side] += d; dims_all.push_back(d); }
    DevBuf<double> rho, U, w;
    RN_TRY(rho.alloc((size_t)(tot[0] + tot[1]))); RN_TRY(U.alloc((size_t)(tot[0] + tot[1]))); RN_TRY(w.alloc((size_t)(wtot[0] + wtot[1])));
    RNT(3, st);
    int rc = density_matrix(p, x, 0, rho.p, st);                                       // line 5
    if (rc == DMRG_OK) rc = density_matrix(p, x, 1, rho.p + tot[0], st);
    RNT(4, st);
    if (rc == DMRG_OK) rc = sector_eig((int)dims_all.size(), dims_all.data(), rho.p, U.p, w.p, st);      // line 6
    RNT(5, st);
    if (rc != DMRG_OK) return rc;
    std::vector<double> wh((size_t)(wtot[0] + wtot[1]));
    RN_TRY(cudaMemcpyAsync(wh.data(), w.p, sizeof(double) * wh.size(), cudaMemcpyDeviceToHost, st));
    RN_TRY(cudaStreamSynchronize(st));
    for (int side = 0; side < 2; side++) {
        const DevBlock &b = *bs[side]; DevBlock &out = *outs[side];
        const int ns = (int)b.dims.size();
        const double *Us = U.p + (side ? tot[0] : 0);
        std::vector<int> keep(ns);
        select_states(ns, b.dims.data(), wh.data() + (side ? wtot[0] : 0), m, keep.data(), disc[side]);  // line 7: which states
        out.labels = b.labels; out.dims = keep; out.n_sites = b.n_sites;
        for (int which = 0; which < 3; which++) {                                // line 7: rotate H, Sz, Sp
            const DevOp &o = which == 0 ? b.H : (which == 1 ? b.Sz : b.Sp);
            DevOp &r = which == 0 ? out.H : (which == 1 ? out.Sz : out.Sp);
            const int nb = (int)o.src.size();
            std::vector<long long> ooff(nb); long long elems = 0;
            rc = rotate_op(ns, b.dims.data(), keep.data(), Us, nb, o.src.data(), o.dst.data(), o.off.data(), o.ld.data(), o.data.p, nullptr, ooff.data(), &elems, st);
            if (rc != DMRG_OK) return rc;
            RN_TRY(r.data.alloc((size_t)elems));
            rc = rotate_op(ns, b.dims.data(), keep.data(), Us, nb, o.src.data(), o.dst.data(), o.off.data(), o.ld.data(), o.data.p, r.data.p, ooff.data(), &elems, st);
            if (rc != DMRG_OK) return rc;
            for (int q = 0; q < nb; q++) if (ooff[q] >= 0) { r.add(o.src[q], o.dst[q], keep[o.dst[q]], keep[o.src[q]]); }
        }
    }
    RNT(6, st);
    return DMRG_OK;
}

}  // namespace
}  // namespace dmrg

using namespace dmrg;

extern "C" {

int dmrg_density_matrix(dmrg_handle_t h, const double *x, int32_t side, double *rho_out, void *stream) {
    if (!h) return DMRG_E_INVALID_ARG;
    Plan *p = reinterpret_cast<Plan *>(h);
    if (!x || !rho_out || side < 0 || side > 1) return fail(p, DMRG_E_INVALID_ARG, "density_matrix: NULL pointer or side not in {0, 1}");
    return density_matrix(p, x, side, rho_out, reinterpret_cast<cudaStream_t>(stream));
}

int dmrg_sector_eig(int32_t n_sectors, const int32_t *dims, double *rho, double *U_out, double *w_out, void *stream) {
    if (n_sectors < 0 || !dims || !rho || !U_out || !w_out) return fail(nullptr, DMRG_E_INVALID_ARG, "sector_eig: bad argument");
    return sector_eig(n_sectors, dims, rho, U_out, w_out, reinterpret_cast<cudaStream_t>(stream));
}

int dmrg_select_states(int32_t n_sectors, const int32_t *dims, const double *w_host, int32_t m, int32_t *m_keep, double *discarded) {
    if (n_sectors < 0 || !dims || !w_host || !m_keep || m < 0) return fail(nullptr, DMRG_E_INVALID_ARG, "select_states: bad argument");
    select_states(n_sectors, dims, w_host, m, m_keep, discarded);
    return DMRG_OK;
}

int dmrg_rotate_op(int32_t n_sectors, const int32_t *dims, const int32_t *m_keep, const double *U, const dmrg_block_op *op,
                   double *out_data, int64_t *out_offset, int64_t *out_elems, void *stream) {
    if (n_sectors < 0 || !dims || !m_keep || !U || !op) return fail(nullptr, DMRG_E_INVALID_ARG, "rotate_op: bad argument");
    std::vector<long long> off(op->offset, op->offset + op->n_blocks), oo(op->n_blocks);
    long long elems = 0;
    int rc = rotate_op(n_sectors, dims, m_keep, U, op->n_blocks, op->src, op->dst, off.data(), op->ld, op->data, out_data, oo.data(), &elems,
                       reinterpret_cast<cudaStream_t>(stream));
    if (out_offset) for (int b = 0; b < op->n_blocks; b++) out_offset[b] = oo[b];
    if (out_elems) *out_elems = elems;
    return rc;
}

int dmrg_infinite_heisenberg(const dmrg_idmrg_options *o, int32_t max_records, int32_t *n_records, int32_t *n_sites, double *energy,
                             double *discarded_left, double *discarded_right, int64_t *target_dim, int32_t *davidson_iters,
                             void *stream) {
    if (!o || !n_records || max_records < 1 || o->n_sites < 4 || o->n_sites % 2 || o->m_keep < 1)
        return fail(nullptr, DMRG_E_INVALID_ARG, "infinite_heisenberg: need an even n_sites >= 4, m_keep >= 1 and room for the records");
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    DevBlock L, R;
    int rc = single_site(L, st); if (rc == DMRG_OK) rc = single_site(R, st);
    *n_records = 0;
    g_tdbg = getenv("DMRG_PLAN_TIMING") != nullptr; g_tl = rn_now(); for (double &v : g_t) v = 0;
    while (rc == DMRG_OK) {
        DevBlock Le, Re;
        RNT(7, st);
        rc = enlarge(L, 0, o->J, o->Delta, Le, st); if (rc != DMRG_OK) break;                  // line 2
        rc = enlarge(R, 1, o->J, o->Delta, Re, st); if (rc != DMRG_OK) break;
        RNT(0, st);
        dmrg_problem pr; memset(&pr, 0, sizeof(pr));
        const int32_t target = 0;
        pr.model = DMRG_HEISENBERG; pr.J = o->J; pr.Delta = o->Delta;
        pr.left = {1, (int32_t)Le.dims.size(), Le.labels.data(), Le.dims.data()};
        pr.right = {1, (int32_t)Re.dims.size(), Re.labels.data(), Re.dims.data()};
        pr.H_L = Le.H.view(); pr.Sz_L = Le.Sz.view(); pr.Sp_L = Le.Sp.view();
        pr.H_R = Re.H.view(); pr.Sz_R = Re.Sz.view(); pr.Sp_R = Re.Sp.view();
        pr.target = &target;
        dmrg_options opt; memset(&opt, 0, sizeof(opt));
        opt.k_max = o->k_max > 0 ? o->k_max : 20; opt.tol = o->tol > 0 ? o->tol : 1e-10; opt.max_iter = o->max_iter > 0 ? o->max_iter : 4000;
        // (reading A16: on a tiny target sector, where k_max is a large fraction of n, ONE Gram-Schmidt pass loses the orthogonality of
        // the basis and Alg. 3 stalls -- the oracle's textbook Davidson does the same; the first superblocks get the second pass)
        long long mL = 0, mR = 0;
        for (int d : Le.dims) mL += d;
        for (int d : Re.dims) mR += d;
        opt.reorth = (mL * mR <= 4096) ? 2 : 1; opt.seed = 1; opt.check_every = 8; opt.reserve_basis = 1;      // (the driver's basis inside the plan's one allocation)
        dmrg_handle_t h = nullptr;
        rc = dmrg_plan_create(&pr, &opt, &h); if (rc != DMRG_OK) break;
        Plan *p = reinterpret_cast<Plan *>(h);
        RNT(1, st);
        DevBuf<double> x; cudaError_t ce = x.alloc((size_t)p->n);
        double lam = 0, rho = 0; int32_t it = 0;
        if (ce != cudaSuccess) { dmrg_plan_destroy(h); return fail(nullptr, DMRG_E_ALLOC, "infinite_heisenberg: eigenvector"); }
        rc = dmrg_lowest_eigenpair(h, nullptr, 1, x.p, &lam, &rho, &it, stream);               // line 3 (start e_argmin(D))
        if (rc == DMRG_NOT_CONVERGED) rc = fail(nullptr, DMRG_E_NUMERIC, "infinite_heisenberg: Davidson did not converge");
        RNT(2, st);
        double dl = 0, dr = 0; DevBlock Ln, Rn;
        if (rc == DMRG_OK) rc = renormalise_both(p, Le, Re, x.p, o->m_keep, Ln, Rn, &dl, &dr, st);      // lines 4-7, both blocks
        const long long n = p->n;
        dmrg_plan_destroy(h);
        if (rc != DMRG_OK) break;
        const int q = *n_records;
        if (q < max_records) {
            if (n_sites) n_sites[q] = Le.n_sites + Re.n_sites;
            if (energy) energy[q] = lam;
            if (discarded_left) discarded_left[q] = dl;
            if (discarded_right) discarded_right[q] = dr;
            if (target_dim) target_dim[q] = n;
            if (davidson_iters) davidson_iters[q] = it;
            *n_records = q + 1;
        }
        if (Le.n_sites + Re.n_sites >= o->n_sites || q + 1 >= max_records) break;
        std::swap(L.labels, Ln.labels); std::swap(L.dims, Ln.dims); L.n_sites = Ln.n_sites;
        std::swap(R.labels, Rn.labels); std::swap(R.dims, Rn.dims); R.n_sites = Rn.n_sites;
        for (int w = 0; w < 3; w++) {
            DevOp &a = w == 0 ? L.H : (w == 1 ? L.Sz : L.Sp), &an = w == 0 ? Ln.H : (w == 1 ? Ln.Sz : Ln.Sp);
            DevOp &b = w == 0 ? R.H : (w == 1 ? R.Sz : R.Sp), &bn = w == 0 ? Rn.H : (w == 1 ? Rn.Sz : Rn.Sp);
            a.src.swap(an.src); a.dst.swap(an.dst); a.ld.swap(an.ld); a.off.swap(an.off); std::swap(a.data.p, an.data.p); std::swap(a.data.n, an.data.n); std::swap(a.elems, an.elems);
            b.src.swap(bn.src); b.dst.swap(bn.dst); b.ld.swap(bn.ld); b.off.swap(bn.off); std::swap(b.data.p, bn.data.p); std::swap(b.data.n, bn.data.n); std::swap(b.elems, bn.elems);
        }
    }
    if (g_tdbg) fprintf(stderr, "idmrg ms: enlarge %.1f plan %.1f davidson %.1f alloc %.1f density %.1f sector_eig %.1f select+rotate %.1f other %.1f\n", g_t[0], g_t[1], g_t[2], g_t[3], g_t[4], g_t[5], g_t[6], g_t[7]);
    return rc;
}

}  // extern "C"
