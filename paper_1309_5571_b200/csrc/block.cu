// block.cu -- block Davidson (Davidson-Liu) for the lowest nb <= 4 eigenpairs: the "block extension ... where more than one
// candidate vectors are added at once resulting in BLAS level 3 operations" of PAPER.md:L247, in the line order of the
// paper's Alg. 3 (L201-237) with b columns wherever Alg. 3 has one (readings A29-A32; oracle/block_davidson.py).
//
// What changes against the single-vector path (davidson.cu):
//   line 2   the na newest basis vectors are projected by ONE grouped launch (gemm.cu, ticket = unit * nrhs + rhs);
//   line 3   G(:, new) = V^T W(:, new): one pass over V serves all na columns (bvtw_kernel: a warp keeps an 8 x na block of
//            accumulators, V is read once);
//   line 4   the nb lowest eigenpairs of the k x k matrix (parallel cyclic Jacobi, one CTA);
//   5-10     X = V Y, W Y, R, ||r_i||, T = R / g(theta_i - D): one pass over V and W for all nb pairs;
//   12-13    S = V^T T, T -= V S: one pass each for all active columns; the b x b Gram matrix of T comes with the pass;
//   14       the corrections are orthonormalised among themselves by Cholesky QR applied twice (the unique thin QR factor
//            with positive diagonal, reading A32; two passes bring ||Q^T Q - I|| to rounding level).
// All reductions have a fixed order (per-CTA partials, last CTA sums them in index order): bitwise reproducible.
#include <cmath>
#include <cstring>
#include "internal.h"

namespace dmrg {

namespace {

constexpr int BT = 256;                       // threads per CTA of the streaming kernels
constexpr int BPS = KMAX * BMAX + 16;         // partials row: [rhs][column] dot products, then 16 scalars
constexpr double GUARD = 1e-8;                // A14

struct Cols { int c[BMAX]; };                 // active correction columns (indices into the T buffer)

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ bool last_block_arrives(int *counter) {
    __shared__ int s_last;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        int old = atomicAdd(counter, 1);
        s_last = (old == (int)gridDim.x - 1);
        if (s_last) *counter = 0;
    }
    __syncthreads();
    if (s_last) __threadfence();
    return s_last != 0;
}
// sum over CTAs of partials column `col`, in CTA order (thread-private chain: fixed order)
__device__ __forceinline__ double sum_column(const double *partials, int col, int nblocks) {
    double a0 = 0.0, a1 = 0.0;
    int b = 0;
    for (; b + 1 < nblocks; b += 2) { a0 += __ldcg(partials + (long long)b * BPS + col); a1 += __ldcg(partials + (long long)(b + 1) * BPS + col); }
    if (b < nblocks) a0 += __ldcg(partials + (long long)b * BPS + col);
    return a0 + a1;
}

// ------------------------------------------------------------------ line 3 / 12: out[r][j] = V(:,j)^T Z(:,cols[r])
// Warp w of the CTA owns the column chunk 8 (w mod nch) .. +7 (nch = ceil(kk / 8)) and the row group w / nch; a lane walks
// row pairs (16-byte loads).  V is read exactly once from HBM; the na columns of Z are re-read by the nch chunk warps of a
// CTA out of L1.
template <int VEC>
__global__ void __launch_bounds__(BT)
bvtw_kernel(const double *__restrict__ V, long long ldv, int kk, const double *__restrict__ Z, long long ldz, Cols cols, int na,
            long long n, double *__restrict__ partials, int *counter, double *__restrict__ out) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int nch = (kk + 7) >> 3;
    const int groups = (BT / 32) / nch;                 // row groups per CTA
    const int ch = warp % nch, rg = warp / nch;
    double acc[8][BMAX];
#pragma unroll
    for (int q = 0; q < 8; q++)
#pragma unroll
        for (int r = 0; r < BMAX; r++) acc[q][r] = 0.0;
    if (rg < groups) {
        const int j0 = ch * 8;
        const long long stride = (long long)gridDim.x * groups * 32 * VEC;
        for (long long p = (((long long)blockIdx.x * groups + rg) * 32 + lane) * VEC; p < n; p += stride) {
            if (VEC == 2 && p + 1 < n) {
                double2 z[BMAX], v[8];
#pragma unroll
                for (int r = 0; r < BMAX; r++) if (r < na) z[r] = *reinterpret_cast<const double2 *>(Z + cols.c[r] * ldz + p);
#pragma unroll
                for (int q = 0; q < 8; q++) if (j0 + q < kk) v[q] = *reinterpret_cast<const double2 *>(V + (j0 + q) * ldv + p);
#pragma unroll
                for (int q = 0; q < 8; q++)
                    if (j0 + q < kk) {
#pragma unroll
                        for (int r = 0; r < BMAX; r++) if (r < na) acc[q][r] = fma(v[q].y, z[r].y, fma(v[q].x, z[r].x, acc[q][r]));
                    }
            } else {
                for (int e = 0; e < VEC && p + e < n; e++) {
#pragma unroll
                    for (int q = 0; q < 8; q++)
                        if (j0 + q < kk) {
                            const double v = V[(j0 + q) * ldv + p + e];
#pragma unroll
                            for (int r = 0; r < BMAX; r++) if (r < na) acc[q][r] = fma(v, Z[cols.c[r] * ldz + p + e], acc[q][r]);
                        }
                }
            }
        }
    }
    __shared__ double s_acc[BT / 32][8 * BMAX];
#pragma unroll
    for (int q = 0; q < 8; q++)
#pragma unroll
        for (int r = 0; r < BMAX; r++) {
            const double v = warp_sum(acc[q][r]);
            if (lane == 0) s_acc[warp][q * BMAX + r] = v;
        }
    __syncthreads();
    // CTA partial of (rhs r, column j): the row groups of chunk j / 8 in group order
    if (threadIdx.x < KMAX * BMAX) {
        const int r = threadIdx.x / KMAX, j = threadIdx.x % KMAX;
        double v = 0.0;
        if (j < kk && r < na)
            for (int g = 0; g < groups; g++) v += s_acc[g * nch + (j >> 3)][(j & 7) * BMAX + r];
        partials[(long long)blockIdx.x * BPS + threadIdx.x] = v;
    }
    if (!last_block_arrives(counter)) return;
    if (threadIdx.x < KMAX * BMAX) {
        const int r = threadIdx.x / KMAX, j = threadIdx.x % KMAX;
        if (j < kk && r < na) out[r * KMAX + j] = sum_column(partials, threadIdx.x, gridDim.x);
    }
}

// ------------------------------------------------------------------ lines 5-10 for nb pairs in one pass over V and W
__global__ void __launch_bounds__(BT)
bresidual_kernel(const double *__restrict__ V, const double *__restrict__ W, long long ldv, int k, const double *__restrict__ D,
                 long long n, BlockState *st, int nb, double *__restrict__ T, double *__restrict__ XS, double *__restrict__ WS,
                 long long ldt, int write_xw, double *__restrict__ partials, int *counter) {
    __shared__ double s_y[KMAX][BMAX];
    __shared__ double s_th[BMAX];
    for (int e = threadIdx.x; e < KMAX * BMAX; e += BT) s_y[e / BMAX][e % BMAX] = (e / BMAX < k && e % BMAX < nb) ? st->Y[e] : 0.0;
    if (threadIdx.x < BMAX) s_th[threadIdx.x] = st->theta[threadIdx.x];
    __syncthreads();
    double rho2[BMAX], nx2[BMAX];
#pragma unroll
    for (int r = 0; r < BMAX; r++) { rho2[r] = 0.0; nx2[r] = 0.0; }
    for (long long p = (long long)blockIdx.x * BT + threadIdx.x; p < n; p += (long long)gridDim.x * BT) {
        double x[BMAX], wy[BMAX];
#pragma unroll
        for (int r = 0; r < BMAX; r++) { x[r] = 0.0; wy[r] = 0.0; }
        for (int j = 0; j < k; j++) {
            const double v = V[j * ldv + p], w = W[j * ldv + p];
#pragma unroll
            for (int r = 0; r < BMAX; r++) { x[r] = fma(v, s_y[j][r], x[r]); wy[r] = fma(w, s_y[j][r], wy[r]); }
        }
        const double d = D[p];
#pragma unroll
        for (int r = 0; r < BMAX; r++)
            if (r < nb) {
                const double res = wy[r] - s_th[r] * x[r];
                rho2[r] = fma(res, res, rho2[r]);
                double g = s_th[r] - d;
                if (fabs(g) < GUARD) g = copysign(GUARD, g);
                T[r * ldt + p] = res / g;
                if (write_xw) { XS[r * ldt + p] = x[r]; WS[r * ldt + p] = wy[r]; nx2[r] = fma(x[r], x[r], nx2[r]); }
            }
    }
    __shared__ double s_r[BT / 32][2 * BMAX];
#pragma unroll
    for (int r = 0; r < BMAX; r++) {
        const double a = warp_sum(rho2[r]), b = warp_sum(nx2[r]);
        if ((threadIdx.x & 31) == 0) { s_r[threadIdx.x >> 5][r] = a; s_r[threadIdx.x >> 5][BMAX + r] = b; }
    }
    __syncthreads();
    if (threadIdx.x < 2 * BMAX) {
        double v = 0.0;
        for (int q = 0; q < BT / 32; q++) v += s_r[q][threadIdx.x];
        partials[(long long)blockIdx.x * BPS + KMAX * BMAX + threadIdx.x] = v;
    }
    if (!last_block_arrives(counter)) return;
    if (threadIdx.x < 2 * BMAX) {
        const double a = sum_column(partials, KMAX * BMAX + threadIdx.x, gridDim.x);
        if (threadIdx.x < BMAX) st->rho2[threadIdx.x] = a; else st->nx2[threadIdx.x - BMAX] = a;
    }
}

// ------------------------------------------------------------------ line 13 for the active columns + their Gram matrix
__global__ void __launch_bounds__(BT)
bsub_kernel(const double *__restrict__ V, long long ldv, int kk, const double *__restrict__ S, double *__restrict__ T, long long ldt,
            Cols cols, int na, long long n, double *__restrict__ partials, int *counter, double *__restrict__ gram) {
    __shared__ double s_s[KMAX][BMAX];
    for (int e = threadIdx.x; e < KMAX * BMAX; e += BT) { const int j = e / BMAX, r = e % BMAX; s_s[j][r] = (j < kk && r < na) ? S[r * KMAX + j] : 0.0; }
    __syncthreads();
    double g[BMAX][BMAX];
#pragma unroll
    for (int a = 0; a < BMAX; a++)
#pragma unroll
        for (int b = 0; b < BMAX; b++) g[a][b] = 0.0;
    for (long long p = (long long)blockIdx.x * BT + threadIdx.x; p < n; p += (long long)gridDim.x * BT) {
        double t[BMAX];
#pragma unroll
        for (int r = 0; r < BMAX; r++) t[r] = r < na ? T[cols.c[r] * ldt + p] : 0.0;
        for (int j = 0; j < kk; j++) {
            const double v = V[j * ldv + p];
#pragma unroll
            for (int r = 0; r < BMAX; r++) t[r] = fma(-v, s_s[j][r], t[r]);
        }
#pragma unroll
        for (int r = 0; r < BMAX; r++) if (r < na) T[cols.c[r] * ldt + p] = t[r];
#pragma unroll
        for (int a = 0; a < BMAX; a++)
#pragma unroll
            for (int b = a; b < BMAX; b++) g[a][b] = fma(t[a], t[b], g[a][b]);
    }
    __shared__ double s_g[BT / 32][BMAX * BMAX];
#pragma unroll
    for (int a = 0; a < BMAX; a++)
#pragma unroll
        for (int b = a; b < BMAX; b++) {
            const double v = warp_sum(g[a][b]);
            if ((threadIdx.x & 31) == 0) s_g[threadIdx.x >> 5][a * BMAX + b] = v;
        }
    __syncthreads();
    if (threadIdx.x < BMAX * BMAX) {
        const int a = threadIdx.x / BMAX, b = threadIdx.x % BMAX;
        double v = 0.0;
        if (b >= a) for (int q = 0; q < BT / 32; q++) v += s_g[q][threadIdx.x];
        partials[(long long)blockIdx.x * BPS + KMAX * BMAX + threadIdx.x] = v;
    }
    if (!last_block_arrives(counter)) return;
    if (threadIdx.x < BMAX * BMAX) gram[threadIdx.x] = sum_column(partials, KMAX * BMAX + threadIdx.x, gridDim.x);
}

// Cholesky of the na x na Gram matrix G = R^T R (R upper, positive diagonal) and Rinv = R^{-1}: T = Q R  =>  Q = T Rinv.
__global__ void bchol_kernel(BlockState *st, int na) {
    if (threadIdx.x != 0) return;
    double R[BMAX][BMAX], Ri[BMAX][BMAX];
    for (int a = 0; a < BMAX; a++) for (int b = 0; b < BMAX; b++) { R[a][b] = 0.0; Ri[a][b] = 0.0; }
    bool bad = false;
    for (int j = 0; j < na; j++) {
        for (int i = 0; i <= j; i++) {
            double s = st->gram[i * BMAX + j];
            for (int m = 0; m < i; m++) s -= R[m][i] * R[m][j];
            if (i == j) {
                if (!(s > 0.0) || isinf(s)) { bad = true; s = 1.0; }
                R[j][j] = sqrt(s);
            } else R[i][j] = s / R[i][i];
        }
    }
    for (int j = 0; j < na; j++) {          // back substitution, column by column of the inverse
        Ri[j][j] = 1.0 / R[j][j];
        for (int i = j - 1; i >= 0; i--) {
            double s = 0.0;
            for (int m = i + 1; m <= j; m++) s -= R[i][m] * Ri[m][j];
            Ri[i][j] = s / R[i][i];
        }
    }
    for (int a = 0; a < BMAX; a++) for (int b = 0; b < BMAX; b++) st->Rinv[a * BMAX + b] = Ri[a][b];
    if (bad) st->error = 1;
}

// out(:,r) = sum_{r' <= r} T(:,cols[r']) Rinv[r'][r]  (+ the Gram matrix of the result, for the second Cholesky-QR pass)
__global__ void __launch_bounds__(BT)
bscale_kernel(const double *T, long long ldt, Cols cols, int na, const BlockState *st, int identity,
              double *out, long long ldo, Cols ocols, long long n, double *__restrict__ partials, int *counter,
              double *__restrict__ gram) {
    __shared__ double s_ri[BMAX][BMAX];
    if (threadIdx.x < BMAX * BMAX) {
        const int a = threadIdx.x / BMAX, b = threadIdx.x % BMAX;
        s_ri[a][b] = identity ? (a == b ? 1.0 : 0.0) : st->Rinv[threadIdx.x];
    }
    __syncthreads();
    double g[BMAX][BMAX];
#pragma unroll
    for (int a = 0; a < BMAX; a++)
#pragma unroll
        for (int b = 0; b < BMAX; b++) g[a][b] = 0.0;
    for (long long p = (long long)blockIdx.x * BT + threadIdx.x; p < n; p += (long long)gridDim.x * BT) {
        double t[BMAX], q[BMAX];
#pragma unroll
        for (int r = 0; r < BMAX; r++) t[r] = r < na ? T[cols.c[r] * ldt + p] : 0.0;
#pragma unroll
        for (int r = 0; r < BMAX; r++) {
            double a = 0.0;
#pragma unroll
            for (int m = 0; m < BMAX; m++) if (m <= r) a = fma(t[m], s_ri[m][r], a);
            q[r] = a;
        }
#pragma unroll
        for (int r = 0; r < BMAX; r++) if (r < na) out[ocols.c[r] * ldo + p] = q[r];
#pragma unroll
        for (int a = 0; a < BMAX; a++)
#pragma unroll
            for (int b = a; b < BMAX; b++) g[a][b] = fma(q[a], q[b], g[a][b]);
    }
    if (!gram) return;
    __shared__ double s_g[BT / 32][BMAX * BMAX];
#pragma unroll
    for (int a = 0; a < BMAX; a++)
#pragma unroll
        for (int b = a; b < BMAX; b++) {
            const double v = warp_sum(g[a][b]);
            if ((threadIdx.x & 31) == 0) s_g[threadIdx.x >> 5][a * BMAX + b] = v;
        }
    __syncthreads();
    if (threadIdx.x < BMAX * BMAX) {
        const int a = threadIdx.x / BMAX, b = threadIdx.x % BMAX;
        double v = 0.0;
        if (b >= a) for (int q = 0; q < BT / 32; q++) v += s_g[q][threadIdx.x];
        partials[(long long)blockIdx.x * BPS + KMAX * BMAX + threadIdx.x] = v;
    }
    if (!last_block_arrives(counter)) return;
    if (threadIdx.x < BMAX * BMAX) gram[threadIdx.x] = sum_column(partials, KMAX * BMAX + threadIdx.x, gridDim.x);
}

// restart (A31): V(:,r) = X_r / ||X_r||, W(:,r) = (W Y)_r / ||X_r||
__global__ void __launch_bounds__(BT)
bcollapse_kernel(double *__restrict__ V, double *__restrict__ W, long long ldv, const double *__restrict__ XS,
                 const double *__restrict__ WS, long long ldt, int nb, long long n, const BlockState *st) {
    double inv[BMAX];
#pragma unroll
    for (int r = 0; r < BMAX; r++) inv[r] = r < nb ? 1.0 / sqrt(st->nx2[r]) : 0.0;
    for (long long p = (long long)blockIdx.x * BT + threadIdx.x; p < n; p += (long long)gridDim.x * BT)
#pragma unroll
        for (int r = 0; r < BMAX; r++)
            if (r < nb) { V[r * ldv + p] = XS[r * ldt + p] * inv[r]; if (W) W[r * ldv + p] = WS[r * ldt + p] * inv[r]; }
}
__global__ void bcollapse_small_kernel(BlockState *st, int nb) {
    for (int e = threadIdx.x; e < KMAX * KMAX; e += blockDim.x) st->G[e] = 0.0;
    __syncthreads();
    if (threadIdx.x < nb) st->G[threadIdx.x * KMAX + threadIdx.x] = st->theta[threadIdx.x];
}
__global__ void breset_kernel(BlockState *st) {
    for (int e = threadIdx.x; e < KMAX * KMAX; e += blockDim.x) st->G[e] = 0.0;
    for (int e = threadIdx.x; e < KMAX * BMAX; e += blockDim.x) { st->Y[e] = 0.0; st->S[e] = 0.0; }
    if (threadIdx.x < BMAX) { st->theta[threadIdx.x] = 0.0; st->rho2[threadIdx.x] = 0.0; st->nx2[threadIdx.x] = 0.0; }
    if (threadIdx.x == 0) st->error = 0;
}

// ------------------------------------------------------------------ line 4 for nb pairs
// New columns of G from the dot products in st->S (mirrored, A18), then all eigenpairs of G(0:k,0:k) by parallel cyclic
// Jacobi (one CTA, thread (i,j) owns A(i,j); round-robin ordering: k/2 disjoint rotations per round), then the nb lowest
// (ascending; lowest index on ties), each with the largest-|y_p| component positive (A18) and theta = y^T G y.
__device__ __forceinline__ void rot_cs(double app, double aqq, double apq, double &c, double &s) {
    c = 1.0; s = 0.0;
    if (apq == 0.0) return;
    const double tau = (aqq - app) / (2.0 * apq);
    if (!(fabs(tau) < 1e300)) return;                       // negligible off-diagonal element (or inf/nan)
    const double t = copysign(1.0, tau) / (fabs(tau) + sqrt(fma(tau, tau, 1.0)));
    c = 1.0 / sqrt(fma(t, t, 1.0)); s = t * c;
}
__global__ void __launch_bounds__(1024)
beig_kernel(BlockState *st, int k, int na, int nb) {
    __shared__ double A[KMAX][KMAX + 1], M[KMAX][KMAX + 1], E[KMAX][KMAX + 1], E2[KMAX][KMAX + 1], Gs[KMAX][KMAX + 1];
    __shared__ double s_c[KMAX], s_s[KMAX], s_off[KMAX], s_dg[KMAX];
    __shared__ int s_partner[KMAX], s_isp[KMAX], s_stop, s_pick[BMAX];
    const int tid = threadIdx.x, i = tid >> 5, j = tid & 31;
    const int R = blockDim.x >> 5;
    if (tid < KMAX) { s_partner[tid] = tid; s_isp[tid] = 1; s_c[tid] = 1.0; s_s[tid] = 0.0; }
    // line 3 results: S[r][j] = V(:,j)^T W(:, k-na+r)
    if (i < na && j < k) { const double v = st->S[i * KMAX + j]; st->G[j * KMAX + (k - na + i)] = v; st->G[(k - na + i) * KMAX + j] = v; }
    __syncthreads();
    const bool in = (i < k && j < k);
    const double gij = in ? 0.5 * (st->G[i * KMAX + j] + st->G[j * KMAX + i]) : 0.0;
    A[i][j] = gij; Gs[i][j] = gij; E[i][j] = (i == j) ? 1.0 : 0.0;
    __syncthreads();
    const int n = (k + 1) & ~1;
    if (k > 1) {
        for (int sweep = 0; sweep < 40; sweep++) {
            double off = (in && i != j) ? A[i][j] * A[i][j] : 0.0, dg = (in && i == j) ? A[i][j] * A[i][j] : 0.0;
            off = warp_sum(off); dg = warp_sum(dg);
            if (j == 0) { s_off[i] = off; s_dg[i] = dg; }
            __syncthreads();
            if (tid < 32) {
                double so = tid < R ? s_off[tid] : 0.0, sd = tid < R ? s_dg[tid] : 0.0;
                so = warp_sum(so); sd = warp_sum(sd);
                if (tid == 0) s_stop = (so <= 1e-30 * (sd + so)) ? 1 : 0;
            }
            __syncthreads();
            if (s_stop) break;
            for (int round = 0; round < n - 1; round++) {
                if (tid < n / 2) {
                    int p, q;
                    if (tid == 0) { p = n - 1; q = round; }
                    else { p = (round + tid) % (n - 1); q = (round - tid + (n - 1)) % (n - 1); }
                    if (p > q) { int t = p; p = q; q = t; }
                    double c = 1.0, s = 0.0;
                    if (q < k) rot_cs(A[p][p], A[q][q], A[p][q], c, s);
                    s_partner[p] = q; s_partner[q] = p; s_isp[p] = 1; s_isp[q] = 0;
                    s_c[p] = c; s_c[q] = c; s_s[p] = s; s_s[q] = s;
                }
                __syncthreads();
                {
                    const int pj = s_partner[j];
                    const double c = s_c[j], s = s_s[j];
                    double m, e;
                    if (s_isp[j]) { m = c * A[i][j] - s * A[i][pj]; e = c * E[i][j] - s * E[i][pj]; }
                    else          { m = s * A[i][pj] + c * A[i][j]; e = s * E[i][pj] + c * E[i][j]; }
                    M[i][j] = m; E2[i][j] = e;
                }
                __syncthreads();
                {
                    const int pi = s_partner[i];
                    const double c = s_c[i], s = s_s[i];
                    A[i][j] = s_isp[i] ? c * M[i][j] - s * M[pi][j] : s * M[pi][j] + c * M[i][j];
                    E[i][j] = E2[i][j];
                }
                __syncthreads();
            }
        }
    }
    // the nb lowest eigenvalues, ascending, lowest index on ties (selection by rank: fixed, data-independent order of work)
    if (tid < k) {
        int rank = 0;
        for (int q = 0; q < k; q++) if (A[q][q] < A[tid][tid] || (A[q][q] == A[tid][tid] && q < tid)) rank++;
        if (rank < nb) s_pick[rank] = tid;
    }
    __syncthreads();
    if (i < nb) {               // warp i handles pair i
        const int col = s_pick[i];
        double v = j < k ? E[j][col] : 0.0;
        const double nrm = sqrt(warp_sum(v * v));
        double am = fabs(v); int pm = j;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const double a2 = __shfl_xor_sync(0xffffffffu, am, o); const int p2 = __shfl_xor_sync(0xffffffffu, pm, o);
            if (a2 > am || (a2 == am && p2 < pm)) { am = a2; pm = p2; }
        }
        const double vp = __shfl_sync(0xffffffffu, v, pm);
        v *= (vp < 0.0 ? -1.0 : 1.0) / nrm;
        double gv = 0.0;
        for (int m = 0; m < k; m++) {
            const double vm = __shfl_sync(0xffffffffu, v, m);
            if (j < k) gv = fma(Gs[j][m], vm, gv);
        }
        const double th = warp_sum(v * gv);
        st->Y[j * BMAX + i] = j < k ? v : 0.0;
        if (j == 0) st->theta[i] = th;
    }
}

}  // namespace

// ------------------------------------------------------------------ host side
static int bgrid(const Plan *p) { return (int)std::max<long long>(1, std::min<long long>((long long)p->sm_count * 4, (p->n + BT - 1) / BT)); }
static bool al16(const void *q) { return (reinterpret_cast<uintptr_t>(q) & 15) == 0; }

static void launch_bvtw(Plan *p, const double *V, long long ldv, int kk, const double *Z, long long ldz, const Cols &cols, int na,
                        cudaStream_t st) {
    const int grid = std::min(bgrid(p), p->vec_grid);
    if (al16(V) && al16(Z) && ldv % 2 == 0 && ldz % 2 == 0)
        bvtw_kernel<2><<<grid, BT, 0, st>>>(V, ldv, kk, Z, ldz, cols, na, p->n, p->bpartials, p->vec_counter, p->bstate->S);
    else
        bvtw_kernel<1><<<grid, BT, 0, st>>>(V, ldv, kk, Z, ldz, cols, na, p->n, p->bpartials, p->vec_counter, p->bstate->S);
}

static int bcheck(Plan *p, const char *what) {
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? DMRG_OK : fail(p, DMRG_E_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}
static int bread_state(Plan *p, cudaStream_t st) {
    cudaError_t e = cudaMemcpyAsync(p->bstate_host, p->bstate, sizeof(BlockState), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(&p->state_host->gemm_error, &p->state->gemm_error, sizeof(int), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return fail(p, DMRG_E_CUDA, std::string("block state read-back: ") + cudaGetErrorString(e));
    if (p->state_host->gemm_error) return fail(p, DMRG_E_CUDA, "projection: a dependency wait gave up");
    if (p->bstate_host->error) return fail(p, DMRG_E_NUMERIC, "block Davidson breakdown: dependent or non-finite correction vectors");
    return DMRG_OK;
}

// Cholesky QR twice: T(:,cols) -> orthonormal columns written to out(:,ocols) (the Gram matrix of T must be in st->gram)
static void launch_cholqr2(Plan *p, double *T, long long ldt, const Cols &cols, int na, double *out, long long ldo, const Cols &ocols,
                           cudaStream_t st) {
    const int grid = std::min(bgrid(p), p->vec_grid);
    bchol_kernel<<<1, 32, 0, st>>>(p->bstate, na);
    bscale_kernel<<<grid, BT, 0, st>>>(T, ldt, cols, na, p->bstate, 0, T, ldt, cols, p->n, p->bpartials, p->vec_counter, p->bstate->gram);
    bchol_kernel<<<1, 32, 0, st>>>(p->bstate, na);
    bscale_kernel<<<grid, BT, 0, st>>>(T, ldt, cols, na, p->bstate, 0, out, ldo, ocols, p->n, p->bpartials, p->vec_counter, nullptr);
    p->launches += 4;
}

int bdav_init(Plan *p, int nb, const double *X0, long long ldx0, double *V, double *W, long long ldv, cudaStream_t st) {
    (void)W;
    if (!p->bstate) return fail(p, DMRG_E_INVALID_ARG, "block Davidson needs a plan created with options.max_rhs >= 2");
    if (nb < 1 || nb > p->max_rhs || 2 * nb > p->opt.k_max) return fail(p, DMRG_E_INVALID_ARG, "block_init: need 1 <= nb <= max_rhs and 2 nb <= k_max");
    if (!X0 || !V || ldv < p->n || ldx0 < p->n) return fail(p, DMRG_E_INVALID_ARG, "block_init: NULL vectors or a column stride below n");
    const int grid = std::min(bgrid(p), p->vec_grid);
    Cols c; for (int r = 0; r < BMAX; r++) c.c[r] = r;
    breset_kernel<<<1, 256, 0, st>>>(p->bstate);
    // Gram matrix of X0 (identity scaling into the T buffer), then Cholesky QR twice into V(:,0..nb-1)   (A32)
    bscale_kernel<<<grid, BT, 0, st>>>(X0, ldx0, c, nb, p->bstate, 1, p->btvec, p->bld, c, p->n, p->bpartials, p->vec_counter, p->bstate->gram);
    p->launches += 2;
    launch_cholqr2(p, p->btvec, p->bld, c, nb, V, ldv, c, st);
    return bcheck(p, "block_init");
}

// One block iteration (oracle/block_davidson.py: block_step).  Synchronises twice (after the residuals: the host decides
// which pairs are still active and whether the basis restarts; at the end: breakdown flag).
int bdav_step(Plan *p, double *V, double *W, long long ldv, int *k, int *na_io, int nb, double *theta, double *resnorm,
              int *converged, cudaStream_t st) {
    if (!p->bstate) return fail(p, DMRG_E_INVALID_ARG, "block Davidson needs a plan created with options.max_rhs >= 2");
    const int k_max = p->opt.k_max;
    int kk = *k, na = *na_io;
    if (nb < 1 || nb > p->max_rhs || kk < nb || kk > k_max || na < 1 || na > nb || na > kk || ldv < p->n)
        return fail(p, DMRG_E_INVALID_ARG, "block_step: k, na, nb or ldv out of range");
    const int grid = std::min(bgrid(p), p->vec_grid);
    BlockState *S = p->bstate;
    Cols ident; for (int r = 0; r < BMAX; r++) ident.c[r] = r;
    // line 2: the na newest basis vectors through one grouped launch
    double *vnew = V + (long long)(kk - na) * ldv, *wnew = W + (long long)(kk - na) * ldv;
    int rc = apply_H(p, vnew, wnew, nullptr, st, nullptr, na, ldv, ldv);
    if (rc != DMRG_OK) return rc;
    // line 3
    launch_bvtw(p, V, ldv, kk, wnew, ldv, ident, na, st);
    // line 4
    beig_kernel<<<1, 32 * ((kk + 3) / 4 * 4), 0, st>>>(S, kk, na, nb);
    // lines 5-10 (X, W Y kept when the basis may have to restart)
    const int may_restart = (kk + nb > k_max) ? 1 : 0;
    bresidual_kernel<<<grid, BT, 0, st>>>(V, W, ldv, kk, p->D, p->n, S, nb, p->btvec, p->bxs, p->bws, p->bld, may_restart,
                                          p->bpartials, p->vec_counter);
    p->launches += 3;
    rc = bcheck(p, "block_step");
    if (rc == DMRG_OK) rc = bread_state(p, st);
    if (rc != DMRG_OK) return rc;
    const BlockState &h = *p->bstate_host;
    Cols act; int ba = 0;
    for (int r = 0; r < nb; r++) {
        const double rho = sqrt(h.rho2[r]);
        if (theta) theta[r] = h.theta[r];
        if (resnorm) resnorm[r] = rho;
        if (!(rho == rho)) return fail(p, DMRG_E_NUMERIC, "block Davidson breakdown: non-finite residual");
        if (!(rho <= p->opt.tol)) act.c[ba++] = r;
    }
    for (int r = ba; r < BMAX; r++) act.c[r] = 0;
    if (converged) *converged = (ba == 0) ? 1 : 0;
    if (ba == 0) { *na_io = 0; return DMRG_OK; }
    if (kk + ba > k_max) {      // restart (A31)
        bcollapse_kernel<<<grid, BT, 0, st>>>(V, W, ldv, p->bxs, p->bws, p->bld, nb, p->n, S);
        bcollapse_small_kernel<<<1, 256, 0, st>>>(S, nb);
        p->launches += 2;
        kk = nb;
    }
    // lines 12-13 against the basis; the last pass leaves the Gram matrix of the corrections
    for (int pass = 0; pass < p->opt.reorth; pass++) {
        launch_bvtw(p, V, ldv, kk, p->btvec, p->bld, act, ba, st);
        bsub_kernel<<<grid, BT, 0, st>>>(V, ldv, kk, S->S, p->btvec, p->bld, act, ba, p->n, p->bpartials, p->vec_counter, S->gram);
        p->launches += 2;
    }
    // line 14: orthonormalise among themselves, append
    Cols oc; for (int r = 0; r < BMAX; r++) oc.c[r] = kk + r;
    launch_cholqr2(p, p->btvec, p->bld, act, ba, V, ldv, oc, st);
    rc = bcheck(p, "block_step");
    if (rc == DMRG_OK) rc = bread_state(p, st);
    if (rc != DMRG_OK) return rc;
    *k = kk + ba; *na_io = ba;
    return DMRG_OK;
}

// X_out(:,r) = V Y_r / ||V Y_r|| with the Y of the last step
int bdav_ritz(Plan *p, const double *V, const double *W, long long ldv, int k, int nb, double *X_out, long long ldxo, cudaStream_t st) {
    if (!p->bstate || k < 1 || k > p->opt.k_max || nb < 1 || nb > p->max_rhs || ldxo < p->n) return fail(p, DMRG_E_INVALID_ARG, "block_ritz: bad argument");
    const int grid = std::min(bgrid(p), p->vec_grid);
    bresidual_kernel<<<grid, BT, 0, st>>>(V, W, ldv, k, p->D, p->n, p->bstate, nb, p->btvec, p->bxs, p->bws, p->bld, 1, p->bpartials, p->vec_counter);
    bcollapse_kernel<<<grid, BT, 0, st>>>(X_out, nullptr, ldxo, p->bxs, p->bws, p->bld, nb, p->n, p->bstate);
    p->launches += 2;
    return bcheck(p, "block_ritz");
}

int block_alloc(Plan *p) {
    if (p->max_rhs < 2) return DMRG_OK;
    p->bld = (p->n + 15) / 16 * 16;
    const size_t vb = sizeof(double) * (size_t)p->bld * BMAX;
    cudaError_t e = cudaMalloc((void **)&p->bstate, sizeof(BlockState));
    if (e == cudaSuccess) e = cudaMemset(p->bstate, 0, sizeof(BlockState));
    if (e == cudaSuccess) e = cudaMallocHost((void **)&p->bstate_host, sizeof(BlockState));
    if (e == cudaSuccess) e = cudaMalloc((void **)&p->btvec, vb);
    if (e == cudaSuccess) e = cudaMalloc((void **)&p->bxs, vb);
    if (e == cudaSuccess) e = cudaMalloc((void **)&p->bws, vb);
    if (e == cudaSuccess) e = cudaMalloc((void **)&p->bpartials, sizeof(double) * (size_t)p->vec_grid * BPS);
    if (e != cudaSuccess) return fail(p, e == cudaErrorMemoryAllocation ? DMRG_E_ALLOC : DMRG_E_CUDA, std::string("block workspaces: ") + cudaGetErrorString(e));
    memset(p->bstate_host, 0, sizeof(BlockState));
    p->device_bytes += (long long)(sizeof(BlockState) + 3 * vb + sizeof(double) * (size_t)p->vec_grid * BPS);
    cudaFuncAttributes fa;      // load the kernels now (no lazy-loading hiccup in a timed step)
    cudaFuncGetAttributes(&fa, bvtw_kernel<1>); cudaFuncGetAttributes(&fa, bvtw_kernel<2>); cudaFuncGetAttributes(&fa, beig_kernel);
    cudaFuncGetAttributes(&fa, bresidual_kernel); cudaFuncGetAttributes(&fa, bsub_kernel); cudaFuncGetAttributes(&fa, bscale_kernel);
    cudaFuncGetAttributes(&fa, bchol_kernel); cudaFuncGetAttributes(&fa, bcollapse_kernel);
    cudaGetLastError();
    return DMRG_OK;
}
void block_free(Plan *p) {
    cudaFree(p->bstate); if (p->bstate_host) cudaFreeHost(p->bstate_host);
    cudaFree(p->btvec); cudaFree(p->bxs); cudaFree(p->bws); cudaFree(p->bpartials);
}

}  // namespace dmrg
