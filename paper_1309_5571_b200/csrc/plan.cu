// plan.cu -- host planner: admissible sector pairs, operation records grouped by output,
// operator repacking, work units of the grouped launch, diag(H_SB), workspaces.
//
// PAPER.md:L340-342 (operation records; "A, B are fixed" over the Davidson iteration),
// L358-363 (Alg. 5 step 1: records and FLOP workload per output; all records of one output
// stay with one owner -> no merging of outputs), L165-171 (Eq. 11).  The paper's stream
// interleaving (Alg. 6-7) is replaced by ONE grouped launch over ticket-ordered work units: stage-1
// units form the inner product of every two-factor record, stage-2 units form each output tile as
// ONE product whose K dimension is the concatenation over all records of that output (fixed
// order, no atomics); a stage-2 unit waits on the "complete" counter of the T blocks it reads.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <cstdlib>
#include <map>
#include <mutex>
#include "internal.h"
#include <climits>
#include <time.h>

namespace dmrg {

static thread_local std::string g_err;
void set_global_error(const std::string &s) { g_err = s; }
const std::string &global_error() { return g_err; }
int fail(Plan *p, int code, const std::string &msg) {
    if (p) p->err = msg;
    g_err = msg;
    return code;
}

void stream_enter(Plan *p, cudaStream_t st) {
    if (p->last_valid && p->last_stream != st) cudaStreamWaitEvent(st, p->ev_last, 0);
}
void stream_leave(Plan *p, cudaStream_t st) {
    if (p->ev_last) { cudaEventRecord(p->ev_last, st); p->last_stream = st; p->last_valid = true; }
}

// ---------------------------------------------------------------- plan-time kernels
__global__ void repack_kernel(RepackJob j, double *pool) {
    __shared__ double tile[32][33];
    double *dst = pool + j.dst_off;
    const int r0 = blockIdx.y * 32, c0 = blockIdx.x * 32;
    // image address of element (r, c) of the repacked matrix (internal.h: P images [m-tile][k-tile], Q images [n-tile][k-tile])
    const int KT = j.q_role ? (j.rows + BK - 1) / BK : (j.cols + BK - 1) / BK;
    auto at = [&](int r, int c) -> double & {
        if (j.q_role) return dst[((long long)(c / BN) * KT + r / BK) * IMG + img_q_index(r % BK, c % BN)];
        return dst[((long long)(r / BM) * KT + c / BK) * IMG + img_p_index(r % BM, c % BK)];
    };
    if (!j.transpose) {
        for (int rr = threadIdx.y; rr < 32; rr += blockDim.y) {
            int r = r0 + rr, c = c0 + threadIdx.x;
            if (r < j.rows && c < j.cols) {
                double v = j.s1 * j.src1[(long long)r * j.ld1 + c];
                if (j.src2) v += j.s2 * j.src2[(long long)r * j.ld2 + c];
                at(r, c) = v;
            }
        }
    } else {
        // dst(r,c) = src(c,r): read src rows c0.., cols r0..
        for (int rr = threadIdx.y; rr < 32; rr += blockDim.y) {
            int sr = c0 + rr, sc = r0 + threadIdx.x;   // src row, src col
            double v = 0.0;
            if (sr < j.cols && sc < j.rows) {
                v = j.s1 * j.src1[(long long)sr * j.ld1 + sc];
                if (j.src2) v += j.s2 * j.src2[(long long)sr * j.ld2 + sc];
            }
            tile[rr][threadIdx.x] = v;
        }
        __syncthreads();
        for (int rr = threadIdx.y; rr < 32; rr += blockDim.y) {
            int r = r0 + rr, c = c0 + threadIdx.x;
            if (r < j.rows && c < j.cols) at(r, c) = tile[threadIdx.x][rr];
        }
    }
}

__global__ void diag_kernel(DiagJob j, double *D) {
    long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    long long tot = (long long)j.rows * j.cols;
    if (idx >= tot) return;
    int a = (int)(idx / j.cols), b = (int)(idx % j.cols);
    // diagonal elements out of the tile images: A is a P operand (rows x ka), B^T a Q operand (kb x cols)
    double va = j.da ? j.da[((long long)(a / BM) * ((j.ka + BK - 1) / BK) + a / BK) * IMG + img_p_index(a % BM, a % BK)] : 1.0;
    double vb = j.db ? j.db[((long long)(b / BN) * ((j.kb + BK - 1) / BK) + b / BK) * IMG + img_q_index(b % BK, b % BN)] : 1.0;
    D[j.seg_off + idx] += j.c * (va * vb);
}

// ---------------------------------------------------------------- host helpers
namespace {

struct PoolEntry { long long off; int rows, cols; bool q_role; };
struct FactorBlk { int src, dst, entry; };          // entry = pool index
struct Term { bool A_id, B_id; std::vector<FactorBlk> A, B; };
struct Record { int A, B, in_pair, out_pair; };      // pool entries or -1 (identity)
struct TaskHost { uint8_t c_base; long long c_off; int ldc, M, N; int item_begin, item_count; int out_pair; uint8_t c_kind; int axpy_begin = 0, axpy_count = 0; };


struct Builder {
    Plan *p;
    const dmrg_problem *pr;
    std::vector<PoolEntry> pool;
    std::vector<RepackJob> jobs;
    long long pool_elems = 0;
    long long op_elems = 0;

    // q_role: the entry is a right-block factor, stored as B^T = the Q operand (K x N) of its products; left-block
    // factors are P operands (M x K).  Either way the entry is a grid of zero-padded 8 KB tile images.
    int add_entry(bool q_role, const dmrg_block_op &op, int b, const std::vector<int> &dims, bool transpose, double scale,
                  const dmrg_block_op *op2 = nullptr, int b2 = -1, double scale2 = 0.0) {
        int rs = dims[op.dst[b]], cs = dims[op.src[b]];   // source block shape rs x cs
        PoolEntry e;
        e.rows = transpose ? cs : rs;
        e.cols = transpose ? rs : cs;
        e.q_role = q_role;
        e.off = pool_elems;
        pool_elems += q_role ? img_q_elems(e.rows, e.cols) : img_p_elems(e.rows, e.cols);
        op_elems += (long long)e.rows * e.cols;
        RepackJob j{};
        j.src1 = op.data + op.offset[b];
        j.ld1 = op.ld[b];
        j.s1 = scale;
        if (op2) { j.src2 = op2->data + op2->offset[b2]; j.ld2 = op2->ld[b2]; j.s2 = scale2; }
        j.dst_off = e.off; j.rows = e.rows; j.cols = e.cols; j.transpose = transpose ? 1 : 0; j.q_role = q_role ? 1 : 0;
        jobs.push_back(j);
        pool.push_back(e);
        return (int)pool.size() - 1;
    }
};

int check_op(Plan *p, const char *name, const dmrg_block_op &op, const std::vector<int> &dims,
             const std::vector<int> &labs, int nl, bool must_be_diagonal) {
    int ns = (int)dims.size();
    if (op.n_blocks < 0) return fail(p, DMRG_E_INVALID_ARG, std::string(name) + ": n_blocks < 0");
    if (op.n_blocks == 0) return DMRG_OK;
    if (!op.src || !op.dst || !op.offset || !op.ld || !op.data)
        return fail(p, DMRG_E_INVALID_ARG, std::string(name) + ": null array with n_blocks > 0");
    std::vector<int> shift(nl, 0);
    bool have = false;
    for (int b = 0; b < op.n_blocks; b++) {
        int s = op.src[b], d = op.dst[b];
        if (s < 0 || s >= ns || d < 0 || d >= ns)
            return fail(p, DMRG_E_SECTOR, std::string(name) + ": block sector index out of range");
        if (op.ld[b] < dims[s]) return fail(p, DMRG_E_SECTOR, std::string(name) + ": ld smaller than dims[src]");
        if (op.offset[b] < 0) return fail(p, DMRG_E_INVALID_ARG, std::string(name) + ": negative offset");
        if (must_be_diagonal && s != d)
            return fail(p, DMRG_E_SECTOR, std::string(name) + ": must be block-diagonal (src == dst)");
        for (int a = 0; a < nl; a++) {
            int sh = labs[d * nl + a] - labs[s * nl + a];
            if (!have) shift[a] = sh;
            else if (shift[a] != sh)
                return fail(p, DMRG_E_SECTOR, std::string(name) + ": blocks with different label shifts (A4)");
        }
        have = true;
    }
    return DMRG_OK;
}

}  // namespace

// ---------------------------------------------------------------- output sharding
// PAPER.md:L342 "all records of the same output on the same [device]", L362 (Alg. 5 step 1: FLOP workload per output):
// longest-processing-time assignment of the outputs to ranks -- outputs by descending cost (ties: lower index), each to the
// least loaded rank (ties: lower rank).  Pure host arithmetic: every rank computes the same table.
void partition_outputs(int n_outputs, const long long *cost, int n_ranks, int *owner) {
    std::vector<int> ord(n_outputs);
    for (int q = 0; q < n_outputs; q++) ord[q] = q;
    std::stable_sort(ord.begin(), ord.end(), [&](int a, int b) { return cost[a] > cost[b]; });
    std::vector<long long> load(std::max(n_ranks, 1), 0);
    for (int q : ord) {
        int best = 0;
        for (int r = 1; r < n_ranks; r++) if (load[r] < load[best]) best = r;
        owner[q] = best; load[best] += cost[q];
    }
}

// ---------------------------------------------------------------- plan_build
#define CUDA_TRY(p, x) do { cudaError_t e__ = (x); if (e__ != cudaSuccess) { \
    plan_free(p); return fail(nullptr, (e__ == cudaErrorMemoryAllocation) ? DMRG_E_ALLOC : DMRG_E_CUDA, \
    std::string(#x) + ": " + cudaGetErrorString(e__)); } } while (0)

template <class T>
static cudaError_t dev_alloc(Plan *p, T **ptr, long long count) {
    // One device allocation per plan: the buffers are RESERVED here (256-byte aligned slices of one arena) and get their
    // addresses in arena_commit -- a plan is created per superblock, and two dozen cudaMalloc / cudaFree pairs were a third of
    // the time of plan creation + destruction (8.6 + 3.2 ms at cfg 3).
    const size_t bytes = ((size_t)std::max<long long>(count, 1) * sizeof(T) + 255) & ~(size_t)255;
    *ptr = nullptr;
    p->arena_reqs.push_back({reinterpret_cast<void **>(ptr), bytes});
    p->device_bytes += (long long)bytes;
    return cudaSuccess;
}
static cudaError_t arena_commit(Plan *p) {
    size_t total = 0;
    for (auto &r : p->arena_reqs) total += r.second;
    cudaError_t e = cudaMalloc(&p->arena, std::max<size_t>(total, 256));
    if (e != cudaSuccess) return e;
    char *base = static_cast<char *>(p->arena);
    for (auto &r : p->arena_reqs) { *r.first = base; base += r.second; }
    p->arena_reqs.clear();
    return cudaSuccess;
}
// pinned host copies of the Davidson state are recycled across plans (cudaMallocHost costs ~1 ms)
static std::mutex g_state_mu;
static std::vector<DavState *> g_state_free;
static cudaError_t state_host_get(DavState **out) {
    {
        std::lock_guard<std::mutex> lk(g_state_mu);
        if (!g_state_free.empty()) { *out = g_state_free.back(); g_state_free.pop_back(); return cudaSuccess; }
    }
    return cudaHostAlloc((void **)out, sizeof(DavState), cudaHostAllocPortable);
}
static void state_host_put(DavState *s) {
    if (!s) return;
    std::lock_guard<std::mutex> lk(g_state_mu);
    if (g_state_free.size() < 8) g_state_free.push_back(s); else cudaFreeHost(s);
}

static double now_ms() { timespec ts; clock_gettime(CLOCK_MONOTONIC, &ts); return ts.tv_sec * 1e3 + ts.tv_nsec * 1e-6; }
#define TCK(lab) do { if (tdbg) { double t = now_ms(); fprintf(stderr, "  plan %-28s %.3f ms\n", lab, t - tlast); tlast = t; } } while (0)
int plan_build(const dmrg_problem *pr, const dmrg_options *opts, Plan **out, const dmrg_problem_l11r *l11) {
    const bool tdbg = getenv("DMRG_PLAN_TIMING") != nullptr; double tlast = now_ms();
    *out = nullptr;
    if (!pr) return fail(nullptr, DMRG_E_INVALID_ARG, "problem is NULL");
    if (pr->model != DMRG_HEISENBERG && pr->model != DMRG_HUBBARD)
        return fail(nullptr, DMRG_E_INVALID_ARG, "unknown model");
    const int nl = pr->left.n_labels;
    if (nl < 1 || nl > 2 || pr->right.n_labels != nl)
        return fail(nullptr, DMRG_E_INVALID_ARG, "n_labels must be 1 or 2 and equal on both sides");
    if (pr->model == DMRG_HUBBARD && nl != 2)
        return fail(nullptr, DMRG_E_INVALID_ARG, "Hubbard needs two labels (N_up, N_dn)");
    if (pr->left.n_sectors < 0 || pr->right.n_sectors < 0 || !pr->target)
        return fail(nullptr, DMRG_E_INVALID_ARG, "bad sector count or NULL target");
    if ((pr->left.n_sectors && (!pr->left.labels || !pr->left.dims)) ||
        (pr->right.n_sectors && (!pr->right.labels || !pr->right.dims)))
        return fail(nullptr, DMRG_E_INVALID_ARG, "NULL sector arrays");

    Plan *p = new Plan();
    p->model = pr->model; p->J = pr->J; p->Delta = pr->Delta; p->t = pr->t; p->U = pr->U;
    p->n_labels = nl;
    if (opts) p->opt = *opts;
    else { p->opt.k_max = 20; p->opt.tol = 1e-10; p->opt.max_iter = 2000; p->opt.reorth = 1; p->opt.seed = 1; }
    if (p->opt.k_max == 0) p->opt.k_max = 20;
    if (p->opt.max_iter <= 0) p->opt.max_iter = 2000;
    if (p->opt.reorth <= 0) p->opt.reorth = 1;
    if (p->opt.check_every <= 0) p->opt.check_every = 8;
    if (p->opt.shard_count < 0 || (p->opt.shard_count > 1 && (p->opt.shard_rank < 0 || p->opt.shard_rank >= p->opt.shard_count))) {
        delete p; return fail(nullptr, DMRG_E_INVALID_ARG, "options: need 0 <= shard_rank < shard_count");
    }
    if (p->opt.max_rhs <= 0) p->opt.max_rhs = 1;
    if (p->opt.max_rhs > BMAX) { delete p; return fail(nullptr, DMRG_E_INVALID_ARG, "options: max_rhs must be 1..4"); }
    p->max_rhs = p->opt.max_rhs;
    if (p->opt.k_max < 2 || p->opt.k_max > KMAX || p->opt.reorth > 2 || !(p->opt.tol >= 0.0)) {
        delete p; return fail(nullptr, DMRG_E_INVALID_ARG, "options: need 2 <= k_max <= 32, reorth in {1,2}, tol >= 0");
    }
    const int nL = pr->left.n_sectors, nR = pr->right.n_sectors;
    p->labL.assign(pr->left.labels, pr->left.labels + (size_t)nL * nl);
    p->labR.assign(pr->right.labels, pr->right.labels + (size_t)nR * nl);
    p->dimL.assign(pr->left.dims, pr->left.dims + nL);
    p->dimR.assign(pr->right.dims, pr->right.dims + nR);
    p->target.assign(pr->target, pr->target + nl);
    for (int d : p->dimL) if (d < 0) { delete p; return fail(nullptr, DMRG_E_SECTOR, "negative sector dimension"); }
    for (int d : p->dimR) if (d < 0) { delete p; return fail(nullptr, DMRG_E_SECTOR, "negative sector dimension"); }

    {   // device properties
        int dev = 0, sms = 0;      // (one attribute, not cudaGetDeviceProperties: that call alone takes over a millisecond)
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) {
            cudaGetLastError();
            delete p; return fail(nullptr, DMRG_E_CUDA, "no CUDA device: this library has no CPU fallback");
        }
        p->sm_count = sms;
    }
    TCK("arguments + device query");

    // ---- operator validation (A4, A26)
    struct Chk { const char *nm; const dmrg_block_op *op; bool left; bool diag; };
    const Chk chks[] = {
        {"H_L", &pr->H_L, true, true}, {"H_R", &pr->H_R, false, true},
        {"Sz_L", &pr->Sz_L, true, true}, {"Sp_L", &pr->Sp_L, true, false},
        {"Sz_R", &pr->Sz_R, false, true}, {"Sp_R", &pr->Sp_R, false, false},
        {"Cup_L", &pr->Cup_L, true, false}, {"Cdn_L", &pr->Cdn_L, true, false},
        {"Cup_R", &pr->Cup_R, false, false}, {"Cdn_R", &pr->Cdn_R, false, false},
        {"D_L", &pr->D_L, true, true}, {"D_R", &pr->D_R, false, true}};
    for (const Chk &c : chks) {
        int rc = check_op(nullptr, c.nm, *c.op, c.left ? p->dimL : p->dimR, c.left ? p->labL : p->labR, nl, c.diag);
        if (rc != DMRG_OK) { delete p; return rc; }
    }

    // ---- admissible pairs and flat layout (A1, A5)
    std::map<std::pair<int, int>, int> pair_index;
    std::vector<std::vector<int>> pairs_of_left(nL);
    for (int i = 0; i < nL; i++) for (int k = 0; k < nR; k++) {
        if (p->dimL[i] == 0 || p->dimR[k] == 0) continue;
        bool ok = true;
        for (int a = 0; a < nl; a++) ok = ok && (p->labL[i * nl + a] + p->labR[k * nl + a] == p->target[a]);
        if (!ok) continue;
        pair_index[{i, k}] = (int)p->pairL.size();
        pairs_of_left[i].push_back((int)p->pairL.size());
        p->pairL.push_back(i); p->pairR.push_back(k);
        p->segOff.push_back(p->n);
        p->n += (long long)p->dimL[i] * p->dimR[k];
    }
    if (p->n == 0) { delete p; return fail(nullptr, DMRG_E_SECTOR, "empty target sector (no admissible pair, A26)"); }
    const int P = (int)p->pairL.size();

    // ---- terms (reading A3, A6, A7) -> pool entries
    Builder bl; bl.p = p; bl.pr = pr;
    std::vector<Term> terms;
    auto sector_blocks_by_src = [](const dmrg_block_op &op, int ns) {
        std::vector<std::vector<int>> v(ns);
        for (int b = 0; b < op.n_blocks; b++) v[op.src[b]].push_back(b);
        return v;
    };
    {   // H_L (+ U D_L) (x) I   and   I (x) H_R (+ U D_R)
        for (int side = 0; side < 2; side++) {
            const dmrg_block_op &H = side == 0 ? pr->H_L : pr->H_R;
            const dmrg_block_op &Dd = side == 0 ? pr->D_L : pr->D_R;
            const std::vector<int> &dims = side == 0 ? p->dimL : p->dimR;
            const bool useD = (pr->model == DMRG_HUBBARD) && Dd.n_blocks > 0 && pr->U != 0.0;
            Term t; t.A_id = side == 1; t.B_id = side == 0;
            auto hs = sector_blocks_by_src(H, (int)dims.size());
            auto ds = sector_blocks_by_src(Dd, (int)dims.size());
            for (int s = 0; s < (int)dims.size(); s++) {
                if (dims[s] == 0) continue;
                // several blocks on one sector are summed pairwise at most (one H, one D)
                if (hs[s].size() > 1 || ds[s].size() > 1) {
                    delete p; return fail(nullptr, DMRG_E_SECTOR, "H/D: more than one block on a sector");
                }
                int e = -1;
                const bool tr = side == 1;   // right factors are stored as B^T
                if (!hs[s].empty() && useD && !ds[s].empty())
                    e = bl.add_entry(tr, H, hs[s][0], dims, tr, 1.0, &Dd, ds[s][0], pr->U);
                else if (!hs[s].empty())
                    e = bl.add_entry(tr, H, hs[s][0], dims, tr, 1.0);
                else if (useD && !ds[s].empty())
                    e = bl.add_entry(tr, Dd, ds[s][0], dims, tr, pr->U);
                if (e >= 0) (side == 0 ? t.A : t.B).push_back({s, s, e});
            }
            terms.push_back(std::move(t));
        }
    }
    auto parity_sign = [&](int left_sector) {
        int N = 0;
        for (int a = 0; a < nl; a++) N += p->labL[left_sector * nl + a];
        return (N % 2 == 0) ? 1.0 : -1.0;
    };
    if (pr->model == DMRG_HEISENBERG) {
        const double half = 0.5 * pr->J, zz = pr->J * pr->Delta;
        if (pr->Sp_L.n_blocks && pr->Sp_R.n_blocks && half != 0.0) {
            Term tp; tp.A_id = tp.B_id = false;   // S+_L (x) S-_R
            Term tm; tm.A_id = tm.B_id = false;   // S-_L (x) S+_R
            for (int b = 0; b < pr->Sp_L.n_blocks; b++) {
                int s = pr->Sp_L.src[b], d = pr->Sp_L.dst[b];
                if (!p->dimL[s] || !p->dimL[d]) continue;
                tp.A.push_back({s, d, bl.add_entry(false, pr->Sp_L, b, p->dimL, false, half)});
                tm.A.push_back({d, s, bl.add_entry(false, pr->Sp_L, b, p->dimL, true, half)});
            }
            for (int b = 0; b < pr->Sp_R.n_blocks; b++) {
                int s = pr->Sp_R.src[b], d = pr->Sp_R.dst[b];
                if (!p->dimR[s] || !p->dimR[d]) continue;
                // S-_R block d->s has matrix blk^T, so its B^T is blk as stored
                tp.B.push_back({d, s, bl.add_entry(true, pr->Sp_R, b, p->dimR, false, 1.0)});
                tm.B.push_back({s, d, bl.add_entry(true, pr->Sp_R, b, p->dimR, true, 1.0)});
            }
            terms.push_back(std::move(tp));
            terms.push_back(std::move(tm));
        }
        if (pr->Sz_L.n_blocks && pr->Sz_R.n_blocks && zz != 0.0) {
            Term tz; tz.A_id = tz.B_id = false;
            for (int b = 0; b < pr->Sz_L.n_blocks; b++)
                if (p->dimL[pr->Sz_L.src[b]])
                    tz.A.push_back({pr->Sz_L.src[b], pr->Sz_L.dst[b], bl.add_entry(false, pr->Sz_L, b, p->dimL, false, zz)});
            for (int b = 0; b < pr->Sz_R.n_blocks; b++)
                if (p->dimR[pr->Sz_R.src[b]])
                    tz.B.push_back({pr->Sz_R.src[b], pr->Sz_R.dst[b], bl.add_entry(true, pr->Sz_R, b, p->dimR, true, 1.0)});
            terms.push_back(std::move(tz));
        }
    } else {
        const dmrg_block_op *CL[2] = {&pr->Cup_L, &pr->Cdn_L};
        const dmrg_block_op *CR[2] = {&pr->Cup_R, &pr->Cdn_R};
        for (int sg = 0; sg < 2; sg++) {
            if (!CL[sg]->n_blocks || !CR[sg]->n_blocks || pr->t == 0.0) continue;
            Term t1; t1.A_id = t1.B_id = false;   // -t (c+_L P_L) (x) c_R : sign from the INPUT left sector
            Term t2; t2.A_id = t2.B_id = false;   // -t (P_L c_L) (x) c+_R : sign from the OUTPUT left sector
            for (int b = 0; b < CL[sg]->n_blocks; b++) {
                int s = CL[sg]->src[b], d = CL[sg]->dst[b];
                if (!p->dimL[s] || !p->dimL[d]) continue;
                const double c = -pr->t * parity_sign(s);   // s = input of c+, = output of c
                t1.A.push_back({s, d, bl.add_entry(false, *CL[sg], b, p->dimL, false, c)});
                t2.A.push_back({d, s, bl.add_entry(false, *CL[sg], b, p->dimL, true, c)});
            }
            for (int b = 0; b < CR[sg]->n_blocks; b++) {
                int s = CR[sg]->src[b], d = CR[sg]->dst[b];
                if (!p->dimR[s] || !p->dimR[d]) continue;
                t1.B.push_back({d, s, bl.add_entry(true, *CR[sg], b, p->dimR, false, 1.0)});   // c_R: B^T = blk
                t2.B.push_back({s, d, bl.add_entry(true, *CR[sg], b, p->dimR, true, 1.0)});    // c+_R: B^T = blk^T
            }
            terms.push_back(std::move(t1));
            terms.push_back(std::move(t2));
        }
    }

    // ---- l-1-1-r strategy (Eq. 12-13): the sectors given to this function are the COMPOSITE ones -- left
    // (s, sigma1) at index 2 s + sigma1, right (sigma2, s') at index sigma2 * n_r + s' (down = 0, up = 1) -- and the operator
    // quadruplets A (x) a (x) b (x) B of the Heisenberg chain reduce, sector by sector, to Eq. 11 records on the UN-enlarged
    // block operators: the 2 x 2 site operators have one non-zero element per row, so a (x) b only selects the segment and
    // scales it.  H_l 1 1 1 + bond(l, site 1) is a left-only term with blocks between composite sectors of equal label,
    // 1 1 1 H_r + bond(site 2, r) a right-only term, and the bond between the two sites needs no GEMM at all: scaled copies
    // of input segments into output segments (axpy items, added in the epilogue of the output tile).
    std::vector<std::vector<AxpyItem>> out_axpy;
    if (l11) {
        const int nl_ = l11->left.n_sectors, nr_ = l11->right.n_sectors;
        std::vector<int> dl(l11->left.dims, l11->left.dims + nl_), dr(l11->right.dims, l11->right.dims + nr_);
        const double half = 0.5 * l11->J, zz = l11->J * l11->Delta;
        auto diag_block = [](const dmrg_block_op &op, int s) { for (int b = 0; b < op.n_blocks; b++) if (op.src[b] == s && op.dst[b] == s) return b; return -1; };
        Term tl; tl.A_id = false; tl.B_id = true;
        Term tr; tr.A_id = true; tr.B_id = false;
        for (int side = 0; side < 2; side++) {
            const dmrg_block_op &H = side == 0 ? l11->H_l : l11->H_r, &Sz = side == 0 ? l11->Sz_l : l11->Sz_r, &Sp = side == 0 ? l11->Sp_l : l11->Sp_r;
            const std::vector<int> &dims = side == 0 ? dl : dr;
            const int ns = (int)dims.size();
            auto comp = [&](int s, int sg) { return side == 0 ? 2 * s + sg : sg * ns + s; };
            const bool q = side == 1;          // right factors are Q operands, stored as B^T
            Term &t = side == 0 ? tl : tr;
            std::vector<FactorBlk> &list = side == 0 ? t.A : t.B;
            for (int s = 0; s < ns; s++) {
                if (dims[s] == 0) continue;
                const int hb = diag_block(H, s), zb = diag_block(Sz, s);
                for (int sg = 0; sg < 2; sg++) {     // H_b + J Delta sigma Sz_b on (s, sigma)
                    const double c = zz * (sg - 0.5);
                    int e = -1;
                    if (hb >= 0 && zb >= 0 && c != 0.0) e = bl.add_entry(q, H, hb, dims, q, 1.0, &Sz, zb, c);
                    else if (hb >= 0) e = bl.add_entry(q, H, hb, dims, q, 1.0);
                    else if (zb >= 0 && c != 0.0) e = bl.add_entry(q, Sz, zb, dims, q, c);
                    if (e >= 0) list.push_back({comp(s, sg), comp(s, sg), e});
                }
            }
            if (half != 0.0)
                for (int b = 0; b < Sp.n_blocks; b++) {   // S+_b S-_site: (s, up) -> (s', down), and the transpose back
                    const int s0 = Sp.src[b], s1 = Sp.dst[b];
                    if (!dims[s0] || !dims[s1]) continue;
                    list.push_back({comp(s0, 1), comp(s1, 0), bl.add_entry(q, Sp, b, dims, q, half)});
                    list.push_back({comp(s1, 0), comp(s0, 1), bl.add_entry(q, Sp, b, dims, !q, half)});
                }
        }
        terms.push_back(std::move(tl));
        terms.push_back(std::move(tr));
        // bond site 1 - site 2: X'(s,s1';s2',s') += c X(s,s1;s2,s')
        out_axpy.assign(P, {});
        for (int op = 0; op < P; op++) {
            const int cl = p->pairL[op], cr = p->pairR[op];
            const int s = cl / 2, s1 = cl % 2, s2 = cr / nr_, sp = cr % nr_;
            if (zz != 0.0) out_axpy[op].push_back({p->segOff[op], zz * (s1 - 0.5) * (s2 - 0.5)});
            if (half != 0.0 && s1 != s2) {           // (up, down) <-> (down, up)
                auto it = pair_index.find({2 * s + s2, s1 * nr_ + sp});
                if (it != pair_index.end()) out_axpy[op].push_back({p->segOff[it->second], half});
            }
        }
    }

    // ---- operation records, in term order, grouped later by output
    std::vector<Record> recs;
    for (const Term &t : terms) {
        if (t.B_id) {
            for (const FactorBlk &a : t.A)
                for (int ip : pairs_of_left[a.src]) {
                    auto it = pair_index.find({a.dst, p->pairR[ip]});
                    if (it != pair_index.end()) recs.push_back({a.entry, -1, ip, it->second});
                }
        } else if (t.A_id) {
            for (int ip = 0; ip < P; ip++)
                for (const FactorBlk &b : t.B) {
                    if (b.src != p->pairR[ip]) continue;
                    auto it = pair_index.find({p->pairL[ip], b.dst});
                    if (it != pair_index.end()) recs.push_back({-1, b.entry, ip, it->second});
                }
        } else {
            for (const FactorBlk &a : t.A)
                for (int ip : pairs_of_left[a.src])
                    for (const FactorBlk &b : t.B) {
                        if (b.src != p->pairR[ip]) continue;
                        auto it = pair_index.find({a.dst, b.dst});
                        if (it != pair_index.end()) recs.push_back({a.entry, b.entry, ip, it->second});
                    }
        }
    }

    // ---- output sharding (options.shard_count > 1): this plan projects only the output segments its rank owns
    const std::vector<Record> all_recs = recs;         // diag(H_SB) needs every record on every rank
    p->owner.assign(P, 0);
    if (p->opt.shard_count > 1) {
        std::vector<long long> cost(P, 0);
        for (const Record &r : recs) {
            const long long di = p->dimL[p->pairL[r.in_pair]], dk = p->dimR[p->pairR[r.in_pair]];
            const long long dj = p->dimL[p->pairL[r.out_pair]], dl = p->dimR[p->pairR[r.out_pair]];
            if (r.B < 0) cost[r.out_pair] += 2 * dj * di * dk;
            else if (r.A < 0) cost[r.out_pair] += 2 * di * dk * dl;
            else cost[r.out_pair] += std::min(2 * di * dk * dl + 2 * dj * di * dl, 2 * dj * di * dk + 2 * dj * dk * dl);
        }
        partition_outputs(P, cost.data(), p->opt.shard_count, p->owner.data());
        std::vector<Record> mine;
        for (const Record &r : recs) if (p->owner[r.out_pair] == p->opt.shard_rank) mine.push_back(r);
        recs.swap(mine);
    }

    // ---- stage-1 tasks / stage-2 items; association order by FLOP (A24)
    std::vector<GemmItem> items1, items2;
    std::vector<TaskHost> tasks1, tasks2;
    std::vector<std::vector<GemmItem>> out_items(P);
    long long tws_elems = 0, flops = 0, flops1 = 0;
    int n_gemms = 0;
    auto vec2 = [](long long off, int ld) { return (uint8_t)((off % 2 == 0 && ld % 2 == 0) ? 1 : 0); };
    // the input vector's segments as tile images (both operand roles), rewritten by phase 0 of every apply
    std::vector<long long> xpOff(P), xqOff(P);
    std::vector<XSeg> xsegs;
    int n_xrb = 0;
    long long xp_elems = 0, xq_elems = 0;
    for (int op = 0; op < P; op++) {
        const int di = p->dimL[p->pairL[op]], dk = p->dimR[p->pairR[op]];
        xpOff[op] = xp_elems; xp_elems += img_p_elems(di, dk);
        xqOff[op] = xq_elems; xq_elems += img_q_elems(di, dk);
        xsegs.push_back({p->segOff[op], xpOff[op], xqOff[op], di, dk, n_xrb, 0});
        n_xrb += (di + BK - 1) / BK;
    }
    for (const Record &r : recs) {
        const int i = p->pairL[r.in_pair], k = p->pairR[r.in_pair];
        const int j = p->pairL[r.out_pair], l = p->pairR[r.out_pair];
        const long long di = p->dimL[i], dk = p->dimR[k], dj = p->dimL[j], dl = p->dimR[l];
        const long long xp = xpOff[r.in_pair], xq = xqOff[r.in_pair];
        GemmItem it2{};
        int dep = -1;             // stage-1 task whose T block this record's stage-2 item reads
        if (r.B < 0) {            // A (x) I :  X'_jk += A X_ik
            const PoolEntry &A = bl.pool[r.A];
            it2 = {A.off, xq, (int)di, BASE_POOL, BASE_XQ};
            it2.xdep = 1;
            flops += 2 * dj * di * dk; n_gemms += 1;
        } else if (r.A < 0) {     // I (x) B :  X'_il += X_ik B^T
            const PoolEntry &B = bl.pool[r.B];
            it2 = {xp, B.off, (int)dk, BASE_XP, BASE_POOL};
            it2.xdep = 1;
            flops += 2 * di * dk * dl; n_gemms += 1;
        } else {
            const PoolEntry &A = bl.pool[r.A], &B = bl.pool[r.B];
            const long long f1 = 2 * di * dk * dl + 2 * dj * di * dl;   // T = X B^T ; X' += A T
            const long long f2 = 2 * dj * di * dk + 2 * dj * dk * dl;   // T = A X   ; X' += T B^T
            n_gemms += 2;
            GemmItem it1{};
            TaskHost t1{};
            if (f1 <= f2) {       // T (d_i x d_l) is the Q operand of stage 2 (K = d_i): stored as Q images
                const long long toff = tws_elems; tws_elems += img_q_elems(di, dl);
                it1 = {xp, B.off, (int)dk, BASE_XP, BASE_POOL};
                t1 = {BASE_T, toff, 0, (int)di, (int)dl, 0, 1, 0, C_IMG_Q};
                it2 = {A.off, toff, (int)di, BASE_POOL, BASE_T};
                flops += f1; flops1 += 2 * di * dk * dl;
            } else {              // T (d_j x d_k) is the P operand of stage 2 (K = d_k): stored as P images
                const long long toff = tws_elems; tws_elems += img_p_elems(dj, dk);
                it1 = {A.off, xq, (int)di, BASE_POOL, BASE_XQ};
                t1 = {BASE_T, toff, 0, (int)dj, (int)dk, 0, 1, 0, C_IMG_P};
                it2 = {toff, B.off, (int)dk, BASE_T, BASE_POOL};
                flops += f2; flops1 += 2 * dj * di * dk;
            }
            t1.item_begin = (int)items1.size();
            t1.out_pair = r.out_pair;
            it1.xdep = 1; it1.dep = r.in_pair; it1.dep_need = (int)(di * dk);     // counters: X segments first, T blocks after
            dep = (int)tasks1.size();
            items1.push_back(it1);
            tasks1.push_back(t1);
        }
        if (it2.xdep) { it2.dep = r.in_pair; it2.dep_need = (int)(di * dk); }
        else { it2.dep = P + dep; it2.dep_need = CWARPS * ((tasks1[dep].M + BM - 1) / BM) * ((tasks1[dep].N + BN - 1) / BN); }   // one count per consumer warp
        out_items[r.out_pair].push_back(it2);
    }
    // inside one output the records that read X directly come first in the K order, so that a stage-2 unit
    // starting at k = 0 has work before its first T block is complete (order fixed at plan time: deterministic)
    for (auto &v : out_items)
        std::stable_sort(v.begin(), v.end(), [](const GemmItem &a, const GemmItem &b) { return a.xdep > b.xdep; });
    std::vector<AxpyItem> axpy;
    for (int op = 0; op < P; op++) {
        if (p->opt.shard_count > 1 && p->owner[op] != p->opt.shard_rank) continue;    // not ours: y segment left untouched
        TaskHost t{};
        t.c_base = BASE_Y; t.c_kind = C_ROWMAJOR; t.c_off = p->segOff[op]; t.ldc = p->dimR[p->pairR[op]];
        t.M = p->dimL[p->pairL[op]]; t.N = p->dimR[p->pairR[op]];
        t.item_begin = (int)items2.size(); t.item_count = (int)out_items[op].size(); t.out_pair = op;
        if (!out_axpy.empty()) { t.axpy_begin = (int)axpy.size(); t.axpy_count = (int)out_axpy[op].size(); for (const AxpyItem &a : out_axpy[op]) axpy.push_back(a); }
        for (const GemmItem &it : out_items[op]) items2.push_back(it);
        tasks2.push_back(t);   // outputs without any record are still zero-filled by the kernel
    }

    // ---- work units: tiles x split of the concatenated K (fixed-order second-stage reduce).
    // ONE launch runs both stages; units are handed out through a ticket counter in this order: stage-1 units
    // grouped by output, outputs by descending cost -- so T blocks complete in the order stage 2 consumes them --
    // then the stage-2 units in the same output order, so the last units of the launch are the small ones.
    long long part_elems = 0; int n_counters = 0; int split_tiles2 = 0;
    auto ktiles = [&](const std::vector<GemmItem> &items, const TaskHost &t) {
        int kt = 0;
        for (int q = 0; q < t.item_count; q++) kt += (items[t.item_begin + q].K + BK - 1) / BK;
        return kt;
    };
    auto ntiles = [](const TaskHost &t) { return (long long)((t.M + BM - 1) / BM) * ((t.N + BN - 1) / BN); };
    long long Wtot = 0;
    for (const TaskHost &t : tasks1) Wtot += (long long)ktiles(items1, t) * ntiles(t);
    for (const TaskHost &t : tasks2) Wtot += (long long)ktiles(items2, t) * ntiles(t);
    const int kt_min = 6;
    // target: ~units_per_sm units per SM over the whole apply (DMRG_UNITS_PER_SM overrides for experiments)
    // (measured: 16 is best at cfg 3 / 5a, ~280 k-tile units per SM; 24 at the 4096 sweep, 2200 per SM; flat beyond)
    long long ups = (Wtot / std::max(p->sm_count, 1) < 1000) ? 12 : 24;   // re-measured with the persistent kernel: 10-12 best at cfg 3 / 5a
    if (const char *e = getenv("DMRG_UNITS_PER_SM")) ups = std::max(1, atoi(e));
    // ... but do not aim below kt_floor k-tiles per unit when there is work for it: with little work per SM (the l-1-1-r plans, small superblocks) units of
    // two ring stages are all boundary (l-1-1-r, two blocks of m = 1024: 86 -> 76 us with units of >= 18 k-tiles)
    long long kt_floor = 18;
    if (const char *e = getenv("DMRG_KT_FLOOR")) kt_floor = std::max(1, atoi(e));
    long long kt_unit = std::max<long long>(kt_min, (Wtot + (long long)p->sm_count * ups - 1) / ((long long)p->sm_count * ups));
    if (kt_unit < kt_floor && Wtot / kt_floor >= 4LL * p->sm_count) kt_unit = kt_floor;      // (only if that still leaves two units per CTA)
    std::vector<long long> out_cost(P, 0);
    std::vector<int> unit_out, uo1, uo2;
    // "guided" unit size for stage 2: the outputs that come last in ticket order get smaller K slices (the drain of
    // the launch lasts about one unit, so the last units should be short): scale = clamp(tail * (1 - f), lo, 1) with
    // f = fraction of the stage-2 k-tile volume that precedes the output in ticket order
    std::vector<double> unit_scale(P, 1.0);
    {
        double tail = 3.0, lo = 0.5;     // measured: within 2 % of each other at cfg 3 / 5a / 4096; 3.0 / 0.5 marginally best
        if (const char *e = getenv("DMRG_TAIL")) tail = atof(e);
        if (const char *e = getenv("DMRG_TAIL_LO")) lo = atof(e);
        std::vector<long long> vol(P, 0); long long tot2 = 0;
        std::vector<long long> volall(P, 0);
        for (const TaskHost &t : tasks2) { const int op = t.out_pair; vol[op] = (long long)ktiles(items2, t) * ntiles(t); tot2 += vol[op]; volall[op] = vol[op]; }   // (a sharded plan holds only its own outputs)
        for (const TaskHost &t : tasks1) volall[t.out_pair] += (long long)ktiles(items1, t) * ntiles(t);
        std::vector<int> ord(P);
        for (int op = 0; op < P; op++) ord[op] = op;
        std::stable_sort(ord.begin(), ord.end(), [&](int a, int b) { return volall[a] > volall[b]; });
        long long before = 0;
        for (int op : ord) {
            const double f = tot2 > 0 ? (double)before / (double)tot2 : 0.0;
            if (tail > 0) unit_scale[op] = std::min(1.0, std::max(lo, tail * (1.0 - f)));
            before += vol[op];
        }
    }
    auto make_units = [&](const std::vector<TaskHost> &tasks, const std::vector<GemmItem> &items, int item_shift,
                          bool signals, std::vector<GemmUnit> &units, int *split_tiles) {
        for (size_t ti = 0; ti < tasks.size(); ti++) {
            const TaskHost &t = tasks[ti];
            const int kt = ktiles(items, t);
            const long long kt_unit_t = signals ? kt_unit : std::max<long long>(kt_min, (long long)(kt_unit * unit_scale[t.out_pair]));
            for (int m0 = 0; m0 < t.M; m0 += BM) for (int n0 = 0; n0 < t.N; n0 += BN) {
                int ns = (int)std::max<long long>(1, (kt + kt_unit_t / 2) / kt_unit_t);
                // never split below kt_min k-tiles per unit
                while (ns > 1 && kt / ns < kt_min) ns--;
                int tile_id = -1; long long poff = 0;
                if (ns > 1) { tile_id = n_counters++; poff = part_elems; part_elems += (long long)ns * BM * BN; if (split_tiles) (*split_tiles)++; }
                const int sub = ((std::min(BM, t.M - m0) + 7) / 8) * ((std::min(BN, t.N - n0) + 7) / 8);   // 8x8 sub-tiles with data
                int base = kt / ns, rem = kt % ns, begin = 0;
                for (int sp = 0; sp < ns; sp++) {
                    GemmUnit u{};
                    u.c_off = t.c_off; u.part_off = poff; u.ldc = t.ldc; u.M = t.M; u.N = t.N; u.m0 = m0; u.n0 = n0;
                    u.item_begin = t.item_begin + item_shift; u.item_count = t.item_count;
                    u.kt_begin = begin; u.kt_count = base + (sp < rem ? 1 : 0); begin += u.kt_count;
                    u.tile_id = tile_id; u.split_idx = sp; u.n_split = ns;
                    u.c_base = t.c_base; u.c_kind = t.c_kind; u.c_vec2 = vec2(t.c_off, t.ldc);
                    u.signal = signals ? P + (int)ti : -1;
                    u.cost = u.kt_count * (4 * sub + 64);
                    u.axpy_begin = t.axpy_begin; u.axpy_count = t.axpy_count;
                    {   // resolve kt_begin to (item, k offset) here, so that the kernel does not walk the item list
                        int skip = u.kt_begin, q = 0;
                        for (; q < t.item_count; q++) {
                            const int nkt = (items[t.item_begin + q].K + BK - 1) / BK;
                            if (skip < nkt) break;
                            skip -= nkt;
                        }
                        u.item0 = q; u.k00 = skip * BK;
                    }
                    out_cost[t.out_pair] += u.cost;
                    units.push_back(u);
                    unit_out.push_back(t.out_pair);
                }
            }
        }
    };
    auto order_units = [&](std::vector<GemmUnit> &units, std::vector<int> &uo) {
        std::vector<int> idx(units.size());
        for (size_t q = 0; q < idx.size(); q++) idx[q] = (int)q;
        std::stable_sort(idx.begin(), idx.end(), [&](int a, int b) {
            if (uo[a] != uo[b]) {
                if (out_cost[uo[a]] != out_cost[uo[b]]) return out_cost[uo[a]] > out_cost[uo[b]];
                return uo[a] < uo[b];
            }
            return units[a].cost > units[b].cost;
        });
        // Split K: the LAST slice of a tile in ticket order is its reducer and waits for the other slices.  Slices of one tile
        // are taken within a microsecond of each other and run at different paces (the partner CTA on the SM, edge tiles), so a
        // reducer right behind its siblings idles until the slowest of them is done (measured: 8.4 us per CTA at cfg 3).  The
        // highest slice of every split tile is therefore held back by `lag` tickets: its siblings have then finished
        // (cfg 3 185.0 -> 183.5 us, cfg 5a 186.3 -> 182.7; 75-150 tickets are equivalent, 300 and more lengthen the drain).
        static const int lag = []() { const char *e = getenv("DMRG_REDUCER_LAG"); return e ? atoi(e) : 150; }();
        std::vector<GemmUnit> v; v.reserve(units.size());
        std::vector<std::pair<size_t, int>> held;      // (position at which it is due, unit)
        size_t head = 0;
        for (int q : idx) {
            while (head < held.size() && held[head].first <= v.size()) v.push_back(units[held[head++].second]);
            if (lag > 0 && units[q].n_split > 1 && units[q].split_idx == units[q].n_split - 1) held.push_back({v.size() + (size_t)lag, q});
            else v.push_back(units[q]);
        }
        while (head < held.size()) v.push_back(units[held[head++].second]);
        units.swap(v);
    };
    std::vector<GemmUnit> units1, units2;
    make_units(tasks1, items1, 0, true, units1, nullptr);
    uo1.swap(unit_out);
    make_units(tasks2, items2, (int)items1.size(), false, units2, &split_tiles2);
    uo2.swap(unit_out);
    order_units(units1, uo1);     // out_cost now holds stage 1 + stage 2 of every output
    order_units(units2, uo2);
    std::vector<GemmUnit> units(units1);
    units.insert(units.end(), units2.begin(), units2.end());
    {   // split-K: the slice of a tile that comes LAST in ticket order is its reducer (it waits on smaller tickets only)
        std::vector<int> last_of(n_counters, -1);
        for (size_t q = 0; q < units.size(); q++) if (units[q].tile_id >= 0) last_of[units[q].tile_id] = (int)q;
        for (int t = 0; t < n_counters; t++) if (last_of[t] >= 0) units[last_of[t]].reducer = 1;
    }
    std::vector<GemmItem> items(items1);
    items.insert(items.end(), items2.begin(), items2.end());
    p->n_deps_t = (int)tasks1.size();
    p->n_deps = P + p->n_deps_t;
    // Streamed input (dmrg_davidson_step_host with a pinned v_in): a second copy of the unit list in an order that follows the
    // arrival of x (ascending address): the stage-1 units sorted by the segment they read (each reads exactly one) and by tile
    // row, and the stage-2 units of an output `lag` x SM-count tickets after the last stage-1 unit that reads a segment the
    // output needs.  Same units, tiles, split-K slices and slice order: same bits; waits are on smaller tickets or loaders only.
    std::vector<GemmUnit> units_s;
    {
        static const int s_lag = []() { const char *e = getenv("DMRG_STREAM_LAG"); return e ? atoi(e) : 1; }();
        std::map<long long, int> op_of_coff;
        for (const TaskHost &t : tasks2) op_of_coff[t.c_off] = t.out_pair;
        std::vector<int> key(P, -1);
        for (const Record &r : recs) key[r.out_pair] = std::max(key[r.out_pair], r.in_pair);
        std::vector<int> s1;
        std::vector<std::vector<int>> s2a(P), s2b(P);
        for (size_t q = 0; q < units.size(); q++) {
            const GemmUnit &u = units[q];
            if (u.signal >= 0) { s1.push_back((int)q); continue; }
            const int o = op_of_coff[u.c_off];
            if (u.n_split > 1 && u.split_idx == u.n_split - 1) s2b[o].push_back((int)q); else s2a[o].push_back((int)q);
        }
        auto seg_of = [&](int q) { return items[units[q].item_begin].dep; };      // a stage-1 unit has one item, and it reads X
        std::stable_sort(s1.begin(), s1.end(), [&](int a, int b) {
            if (seg_of(a) != seg_of(b)) return seg_of(a) < seg_of(b);
            const bool pa = items[units[a].item_begin].p_base == BASE_XP, pb = items[units[b].item_begin].p_base == BASE_XP;
            const int ra = pa ? units[a].m0 : 1 << 30, rb = pb ? units[b].m0 : 1 << 30;      // P-role tiles by row; Q-role ones need every row
            return ra < rb;
        });
        std::vector<int> oord(P);
        for (int op = 0; op < P; op++) oord[op] = op;
        std::stable_sort(oord.begin(), oord.end(), [&](int a, int b) { return key[a] < key[b]; });
        auto emit2 = [&](int o) { for (int q : s2a[o]) units_s.push_back(units[q]); for (int q : s2b[o]) units_s.push_back(units[q]); };
        const size_t lag_units = (size_t)std::max(0, s_lag) * (size_t)p->sm_count;
        std::vector<std::pair<size_t, int>> due;
        size_t head = 0, oi = 0;
        for (size_t a = 0; a < s1.size(); a++) {
            const int sg = seg_of(s1[a]);
            // outputs whose last segment lies before this unit's: all their stage-1 units are out
            while (oi < oord.size() && key[oord[oi]] < sg) { due.push_back({units_s.size() + lag_units, oord[oi]}); oi++; }
            while (head < due.size() && due[head].first <= units_s.size()) emit2(due[head++].second);
            units_s.push_back(units[s1[a]]);
        }
        while (oi < oord.size()) { due.push_back({0, oord[oi]}); oi++; }
        while (head < due.size()) emit2(due[head++].second);
        if (units_s.size() != units.size()) return fail(p, DMRG_E_INVALID_ARG, "planner: streamed unit order lost units");
        for (GemmUnit &u : units_s) u.reducer = 0;
        std::vector<int> last_of(n_counters, -1);
        for (size_t q = 0; q < units_s.size(); q++) if (units_s[q].tile_id >= 0) last_of[units_s[q].tile_id] = (int)q;
        for (int t = 0; t < n_counters; t++) if (last_of[t] >= 0) units_s[last_of[t]].reducer = 1;
    }
    // shares of <= 3456 elements inside one segment, segments in the order the units of that list first need them; the
    // loaders count the arrived elements per 16-row block of a segment, the units wait per row block (gemm.cu)
    std::vector<XShare> xshares;
    {
        std::vector<int> first(P, INT_MAX);
        for (size_t q = 0; q < units_s.size(); q++)
            for (int e = 0; e < units_s[q].item_count; e++) {
                const GemmItem &it = items[units_s[q].item_begin + e];
                if (it.xdep) first[it.dep] = std::min(first[it.dep], (int)q);
            }
        std::vector<int> ord(P);
        for (int op = 0; op < P; op++) ord[op] = op;
        std::stable_sort(ord.begin(), ord.end(), [&](int a, int b) { return first[a] < first[b]; });
        const int chunk = 288 * 12;
        for (int op : ord) {
            const long long ne = (long long)xsegs[op].di * xsegs[op].dk;
            for (long long lo = 0; lo < ne; lo += chunk) xshares.push_back({op, (int)lo, (int)std::min<long long>(ne, lo + chunk), 0});
        }
    }

    // ---- device allocations
    // per-apply buffers and counters exist once per right-hand side (options.max_rhs; block Davidson)
    const int R = p->max_rhs;
    p->tws_elems = tws_elems; p->part_elems = part_elems; p->xp_elems = xp_elems; p->xq_elems = xq_elems; p->n_counters = n_counters;
    tws_elems *= R; part_elems *= R; xp_elems *= R; xq_elems *= R; n_counters *= R;
    p->vec_grid = p->sm_count * 8;      // capacity of the partials buffer; each kernel launches one wave of its own (davidson.cu)
    p->n_xsegs = (int)xsegs.size(); p->n_xshares = (int)xshares.size(); p->axpy_count = (int)axpy.size();
    TCK("records, units (host)");
    // (1) every buffer is reserved, (2) one allocation, (3) initial contents
    CUDA_TRY(p, dev_alloc(p, &p->pool, bl.pool_elems));
    CUDA_TRY(p, dev_alloc(p, &p->tws, tws_elems));
    CUDA_TRY(p, dev_alloc(p, &p->part, part_elems));
    CUDA_TRY(p, dev_alloc(p, &p->ximg_p, xp_elems));
    CUDA_TRY(p, dev_alloc(p, &p->ximg_q, xq_elems));
    CUDA_TRY(p, dev_alloc(p, &p->xsegs, (long long)xsegs.size()));
    CUDA_TRY(p, dev_alloc(p, &p->xshares, (long long)xshares.size()));
    p->n_xrb = n_xrb;
    CUDA_TRY(p, dev_alloc(p, &p->xrb, (long long)n_xrb));
    std::vector<int2> xrows;
    for (int op = 0; op < P; op++)
        if (xsegs[op].dk > 0) for (int r0 = 0; r0 < xsegs[op].di; r0 += 8) xrows.push_back(make_int2(op, r0));
    p->n_xrows = (int)xrows.size();
    CUDA_TRY(p, dev_alloc(p, &p->xrows, (long long)xrows.size()));
    CUDA_TRY(p, dev_alloc(p, &p->counters, n_counters));
    CUDA_TRY(p, dev_alloc(p, &p->D, p->n));
    CUDA_TRY(p, dev_alloc(p, &p->items, (long long)items.size()));
    CUDA_TRY(p, dev_alloc(p, &p->units, (long long)units.size()));
    CUDA_TRY(p, dev_alloc(p, &p->units_stream, (long long)units_s.size()));
    CUDA_TRY(p, dev_alloc(p, &p->axpy, (long long)axpy.size()));
    CUDA_TRY(p, dev_alloc(p, &p->ctrl, (long long)CTRL_DEP0 + (long long)p->n_deps * R));
    if (getenv("DMRG_TRACE")) {   // diagnostics: per-unit timeline of the last apply (dmrg_get_unit_trace)
        // 4 words per unit, then 4 words per CTA (phase stamps: entry, X images written, producer released, exit)
        p->trace_units = (int)units.size() * R + 8 * p->sm_count;
        CUDA_TRY(p, dev_alloc(p, &p->trace, 4LL * std::max<long long>(p->trace_units, 1)));
    }
    CUDA_TRY(p, dev_alloc(p, &p->state, 1));            // Davidson scratch
    CUDA_TRY(p, dev_alloc(p, &p->tvec, p->n));
    CUDA_TRY(p, dev_alloc(p, &p->xs, p->n));
    CUDA_TRY(p, dev_alloc(p, &p->ws, p->n));
    CUDA_TRY(p, dev_alloc(p, &p->partials, (long long)p->vec_grid * (KMAX + 2)));
    CUDA_TRY(p, dev_alloc(p, &p->vec_counter, 4));
    if (p->opt.reserve_basis) {                          // the drivers' own basis
        p->ldv_own = (p->n + 15) / 16 * 16;
        CUDA_TRY(p, dev_alloc(p, &p->Vown, p->ldv_own * p->opt.k_max));
        CUDA_TRY(p, dev_alloc(p, &p->Wown, p->ldv_own * p->opt.k_max));
        p->own_basis_in_arena = true;
    }
    {
        cudaError_t ea = arena_commit(p);
        if (ea != cudaSuccess) { std::string m = std::string("device allocation of the plan: ") + cudaGetErrorString(ea); plan_free(p); return fail(nullptr, ea == cudaErrorMemoryAllocation ? DMRG_E_ALLOC : DMRG_E_CUDA, m); }
    }
    TCK("arena cudaMalloc");
    CUDA_TRY(p, cudaMemset(p->ximg_p, 0, sizeof(double) * std::max<long long>(xp_elems, 1)));   // the pads stay zero for good
    CUDA_TRY(p, cudaMemset(p->ximg_q, 0, sizeof(double) * std::max<long long>(xq_elems, 1)));
    if (!xsegs.empty()) CUDA_TRY(p, cudaMemcpy(p->xsegs, xsegs.data(), xsegs.size() * sizeof(XSeg), cudaMemcpyHostToDevice));
    if (!xshares.empty()) CUDA_TRY(p, cudaMemcpy(p->xshares, xshares.data(), xshares.size() * sizeof(XShare), cudaMemcpyHostToDevice));
    if (!axpy.empty()) CUDA_TRY(p, cudaMemcpy(p->axpy, axpy.data(), axpy.size() * sizeof(AxpyItem), cudaMemcpyHostToDevice));
    CUDA_TRY(p, cudaMemset(p->ctrl, 0, sizeof(int) * (CTRL_DEP0 + (size_t)p->n_deps * R)));
    CUDA_TRY(p, cudaMemset(p->xrb, 0, sizeof(int) * (size_t)std::max(n_xrb, 1)));
    if (!xrows.empty()) CUDA_TRY(p, cudaMemcpy(p->xrows, xrows.data(), xrows.size() * sizeof(int2), cudaMemcpyHostToDevice));
    if (p->trace) CUDA_TRY(p, cudaMemset(p->trace, 0, 32 * (size_t)std::max(p->trace_units, 1)));
    CUDA_TRY(p, cudaMemset(p->pool, 0, sizeof(double) * std::max<long long>(bl.pool_elems, 1)));
    CUDA_TRY(p, cudaMemset(p->tws, 0, sizeof(double) * std::max<long long>(tws_elems, 1)));
    CUDA_TRY(p, cudaMemset(p->counters, 0, sizeof(int) * std::max(n_counters, 1)));
    CUDA_TRY(p, cudaMemset(p->D, 0, sizeof(double) * p->n));
    if (!items.empty()) CUDA_TRY(p, cudaMemcpy(p->items, items.data(), items.size() * sizeof(GemmItem), cudaMemcpyHostToDevice));
    if (!units.empty()) CUDA_TRY(p, cudaMemcpy(p->units, units.data(), units.size() * sizeof(GemmUnit), cudaMemcpyHostToDevice));
    if (!units_s.empty()) CUDA_TRY(p, cudaMemcpy(p->units_stream, units_s.data(), units_s.size() * sizeof(GemmUnit), cudaMemcpyHostToDevice));
    p->n_units1 = (int)units1.size(); p->n_units2 = (int)units2.size();
    CUDA_TRY(p, cudaMemset(p->state, 0, sizeof(DavState)));
    CUDA_TRY(p, cudaMemset(p->vec_counter, 0, 4 * sizeof(int)));
    CUDA_TRY(p, state_host_get(&p->state_host));
    memset(p->state_host, 0, sizeof(DavState));

    TCK("memsets + table copies");
    // ---- repack the operators (scaled / transposed / aligned), once
    for (const RepackJob &j : bl.jobs) {
        if (j.rows == 0 || j.cols == 0) continue;
        dim3 grid((j.cols + 31) / 32, (j.rows + 31) / 32), block(32, 8);
        repack_kernel<<<grid, block>>>(j, p->pool);
    }
    CUDA_TRY(p, cudaGetLastError());

    TCK("repack launches");
    // ---- diag(H_SB) (A14): records with (i,k) == (j,l)
    for (const Record &r : all_recs) {
        if (r.in_pair != r.out_pair) continue;
        DiagJob dj{};
        dj.seg_off = p->segOff[r.in_pair];
        dj.rows = p->dimL[p->pairL[r.in_pair]]; dj.cols = p->dimR[p->pairR[r.in_pair]];
        dj.c = 1.0;   // the coefficient is already folded into the left factor
        if (r.A >= 0) { dj.da = p->pool + bl.pool[r.A].off; dj.ka = bl.pool[r.A].cols; }
        if (r.B >= 0) { dj.db = p->pool + bl.pool[r.B].off; dj.kb = bl.pool[r.B].rows; }
        long long tot = (long long)dj.rows * dj.cols;
        diag_kernel<<<(unsigned)((tot + 255) / 256), 256>>>(dj, p->D);
    }
    for (int op = 0; op < P && !out_axpy.empty(); op++)          // l-1-1-r: the diagonal part of the site-site bond
        for (const AxpyItem &a : out_axpy[op]) {
            if (a.x_off != p->segOff[op]) continue;
            DiagJob dj{};
            dj.seg_off = p->segOff[op]; dj.rows = p->dimL[p->pairL[op]]; dj.cols = p->dimR[p->pairR[op]]; dj.c = a.c;
            const long long tot = (long long)dj.rows * dj.cols;
            diag_kernel<<<(unsigned)((tot + 255) / 256), 256>>>(dj, p->D);
        }
    CUDA_TRY(p, cudaGetLastError());

    TCK("diag launches");
    // ---- Davidson scratch
    TCK("davidson scratch alloc");
    CUDA_TRY(p, gemm_kernel_setup());
    TCK("gemm_kernel_setup");
    dav_setup(p);
    TCK("dav_setup");
    // everything a hot call needs exists from here on: side stream and events of dmrg_davidson_step_host, the ordering
    // event, and (options.reserve_basis) the drivers' own basis
    CUDA_TRY(p, cudaStreamCreateWithFlags(&p->side, cudaStreamNonBlocking));
    CUDA_TRY(p, cudaEventCreateWithFlags(&p->ev_apply, cudaEventDisableTiming));
    CUDA_TRY(p, cudaEventCreateWithFlags(&p->ev_side, cudaEventDisableTiming));
    CUDA_TRY(p, cudaEventCreateWithFlags(&p->ev_last, cudaEventDisableTiming));
    { int rcb = block_alloc(p); if (rcb != DMRG_OK) { std::string m = p->err; plan_free(p); return fail(nullptr, rcb, m); } }
    TCK("stream/events/block_alloc");
    CUDA_TRY(p, cudaDeviceSynchronize());
    TCK("device synchronize");

    // ---- stats
    dmrg_stats &s = p->stats;
    s.n = p->n; s.n_pairs = P; s.n_records = (int)recs.size(); s.n_gemms = n_gemms;
    s.flop_per_apply = flops; s.flop_stage1 = flops1; s.flop_stage2 = flops - flops1; s.operator_elems = bl.op_elems; s.apply_bytes = 8 * (bl.op_elems + 2 * p->n);
    s.stage1_units = p->n_units1; s.stage2_units = p->n_units2; s.stage2_split_tiles = split_tiles2;
    s.pool_bytes = 8 * bl.pool_elems;
    s.workspace_bytes = 8 * (tws_elems + part_elems + xp_elems + xq_elems + 3 * p->n + (long long)p->vec_grid * (KMAX + 2));
    s.device_bytes = p->device_bytes;
    s.kernel_launches_per_apply = 1;
    // apply, V^T w, small eig, residual (+ V^T t fused), { V^T t from the second pass on }, t -= V s, append; +3 on a restart step
    s.kernel_launches_per_step = s.kernel_launches_per_apply + 3 + 2 * p->opt.reorth;
    *out = p;
    return DMRG_OK;
}

void plan_free(Plan *p) {
    if (!p) return;
    cudaFree(p->arena);                                  // every plan buffer is a slice of it
    state_host_put(p->state_host);
    if (!p->own_basis_in_arena) { cudaFree(p->Vown); cudaFree(p->Wown); }      // (allocated later by a driver: api.cu)
    block_free(p);
    if (p->timing.created) for (auto &e : p->timing.ev) cudaEventDestroy(e);
    if (p->ev_apply) cudaEventDestroy(p->ev_apply);
    if (p->ev_side) cudaEventDestroy(p->ev_side);
    if (p->ev_last) cudaEventDestroy(p->ev_last);
    for (auto &g : p->graphs) cudaGraphExecDestroy(g.second.exec);
    if (p->side) cudaStreamDestroy(p->side);
    delete p;
}

}  // namespace dmrg
