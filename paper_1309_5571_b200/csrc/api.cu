// api.cu -- the extern "C" surface declared in include/dmrg_b200.h.  Argument checking and
// marshalling only; every step of the path runs in the kernels of gemm.cu / davidson.cu.
#include <cmath>
#include <cstddef>
#include <cstring>
#include <vector>
#include "internal.h"

namespace dmrg { const std::string &global_error(); }
using namespace dmrg;

namespace {
inline Plan *P(dmrg_handle_t h) { return reinterpret_cast<Plan *>(h); }
inline cudaStream_t S(void *s) { return reinterpret_cast<cudaStream_t>(s); }

// full = false copies only the scalars a step reports (lambda ... flags, the tail of DavState: 80 bytes instead of 17 KB)
int read_state(Plan *p, cudaStream_t st, bool full = true) {
    const size_t off = full ? 0 : offsetof(DavState, lambda);
    cudaError_t e = cudaMemcpyAsync(reinterpret_cast<char *>(p->state_host) + off, reinterpret_cast<const char *>(p->state) + off,
                                    sizeof(DavState) - off, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return fail(p, DMRG_E_CUDA, std::string("state read-back: ") + cudaGetErrorString(e));
    if (p->state_host->gemm_error)
        return fail(p, DMRG_E_CUDA, "projection: a dependency wait gave up (launches of one plan interleaved on two streams, or a lost launch)");
    return DMRG_OK;
}
void ensure_timing(Plan *p) {
    if (!p->timing.created) {
        for (auto &e : p->timing.ev) cudaEventCreate(&e);
        p->timing.created = true;
    }
}
}  // namespace

extern "C" {

int dmrg_version(void) { return 100; }

const char *dmrg_last_error(dmrg_handle_t h) {
    if (h) return P(h)->err.c_str();
    return global_error().c_str();
}

int dmrg_plan_create(const dmrg_problem *problem, const dmrg_options *opts, dmrg_handle_t *out) {
    if (!out) return fail(nullptr, DMRG_E_INVALID_ARG, "out is NULL");
    Plan *p = nullptr;
    int rc = plan_build(problem, opts, &p);
    *out = reinterpret_cast<dmrg_handle_t>(p);
    return rc;
}

int dmrg_plan_create_l11r(const dmrg_problem_l11r *pr, const dmrg_options *opts, dmrg_handle_t *out) {
    if (!out) return fail(nullptr, DMRG_E_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (!pr || pr->left.n_labels != 1 || pr->right.n_labels != 1 || pr->left.n_sectors < 0 || pr->right.n_sectors < 0 ||
        (pr->left.n_sectors && (!pr->left.labels || !pr->left.dims)) || (pr->right.n_sectors && (!pr->right.labels || !pr->right.dims)))
        return fail(nullptr, DMRG_E_INVALID_ARG, "l11r problem: NULL or sectors with other than one label");
    const int nl = pr->left.n_sectors, nr = pr->right.n_sectors;
    const dmrg_block_op *ops[6] = {&pr->H_l, &pr->Sz_l, &pr->Sp_l, &pr->H_r, &pr->Sz_r, &pr->Sp_r};
    for (int q = 0; q < 6; q++) {           // block shapes and label shifts (diagonal: 0; S+: +2)
        const dmrg_block_op &o = *ops[q]; const dmrg_sectors &sec = q < 3 ? pr->left : pr->right;
        if (o.n_blocks < 0 || (o.n_blocks && (!o.src || !o.dst || !o.offset || !o.ld || !o.data))) return fail(nullptr, DMRG_E_INVALID_ARG, "l11r problem: bad operator arrays");
        for (int b = 0; b < o.n_blocks; b++) {
            if (o.src[b] < 0 || o.src[b] >= sec.n_sectors || o.dst[b] < 0 || o.dst[b] >= sec.n_sectors) return fail(nullptr, DMRG_E_SECTOR, "l11r problem: block sector index out of range");
            if (o.ld[b] < sec.dims[o.src[b]]) return fail(nullptr, DMRG_E_SECTOR, "l11r problem: ld smaller than dims[src]");
            if (sec.labels[o.dst[b]] - sec.labels[o.src[b]] != ((q % 3 == 2) ? 2 : 0)) return fail(nullptr, DMRG_E_SECTOR, "l11r problem: H, Sz must keep the label, S+ must raise it by 2");
        }
    }
    // composite sectors: left (s, sigma1) at 2 s + sigma1, right (sigma2, s') at sigma2 * n_r + s'   (down = 0 / label -1, up = 1 / +1)
    std::vector<int32_t> labL(2 * nl), dimL(2 * nl), labR(2 * nr), dimR(2 * nr);
    for (int s = 0; s < nl; s++) for (int g = 0; g < 2; g++) { labL[2 * s + g] = pr->left.labels[s] + (g ? 1 : -1); dimL[2 * s + g] = pr->left.dims[s]; }
    for (int g = 0; g < 2; g++) for (int s = 0; s < nr; s++) { labR[g * nr + s] = pr->right.labels[s] + (g ? 1 : -1); dimR[g * nr + s] = pr->right.dims[s]; }
    dmrg_problem lr; memset(&lr, 0, sizeof(lr));
    lr.model = DMRG_HEISENBERG; lr.J = pr->J; lr.Delta = pr->Delta;
    lr.left = {1, 2 * nl, labL.data(), dimL.data()}; lr.right = {1, 2 * nr, labR.data(), dimR.data()};
    lr.target = &pr->target_twice_sz;
    Plan *p = nullptr;
    int rc = plan_build(&lr, opts, &p, pr);
    *out = reinterpret_cast<dmrg_handle_t>(p);
    return rc;
}

int dmrg_plan_destroy(dmrg_handle_t h) {
    if (!h) return DMRG_E_INVALID_ARG;
    cudaDeviceSynchronize();
    plan_free(P(h));
    return DMRG_OK;
}

int dmrg_get_layout(dmrg_handle_t h, int64_t *n, int32_t *n_pairs, int32_t *left_sector, int32_t *right_sector,
                    int64_t *seg_offset) {
    if (!h) return DMRG_E_INVALID_ARG;
    Plan *p = P(h);
    if (n) *n = p->n;
    if (n_pairs) *n_pairs = (int32_t)p->pairL.size();
    for (size_t q = 0; q < p->pairL.size(); q++) {
        if (left_sector) left_sector[q] = p->pairL[q];
        if (right_sector) right_sector[q] = p->pairR[q];
        if (seg_offset) seg_offset[q] = p->segOff[q];
    }
    return DMRG_OK;
}

int dmrg_get_stats(dmrg_handle_t h, dmrg_stats *stats) {
    if (!h || !stats) return DMRG_E_INVALID_ARG;
    P(h)->stats.device_bytes = P(h)->device_bytes;
    P(h)->stats.launches = P(h)->launches;
    *stats = P(h)->stats;
    return DMRG_OK;
}

int dmrg_get_diag(dmrg_handle_t h, double *d_out, void *stream) {
    if (!h || !d_out) return DMRG_E_INVALID_ARG;
    Plan *p = P(h);
    cudaError_t e = cudaMemcpyAsync(d_out, p->D, sizeof(double) * p->n, cudaMemcpyDeviceToDevice, S(stream));
    return e == cudaSuccess ? DMRG_OK : fail(p, DMRG_E_CUDA, cudaGetErrorString(e));
}

int dmrg_apply_H(dmrg_handle_t h, const double *x, double *y, void *stream) {
    if (!h) return DMRG_E_INVALID_ARG;
    Plan *p = P(h);
    if (!x || !y) return fail(p, DMRG_E_INVALID_ARG, "apply_H: NULL vector");
    if ((x <= y && y < x + p->n) || (y <= x && x < y + p->n)) return fail(p, DMRG_E_INVALID_ARG, "apply_H: x and y overlap");
    stream_enter(p, S(stream));
    const int rc = apply_H(p, x, y, nullptr, S(stream));
    stream_leave(p, S(stream));
    return rc;
}

int dmrg_davidson_init(dmrg_handle_t h, const double *x0, int32_t start_at_argmin_diag, double *V, double *W,
                       int64_t ldv, void *stream) {
    if (!h) return DMRG_E_INVALID_ARG;
    Plan *p = P(h);
    if (!V || !W || ldv < p->n) return fail(p, DMRG_E_INVALID_ARG, "davidson_init: NULL basis or ldv < n");
    p->state_host->done = 0;
    stream_enter(p, S(stream));
    const int rc = dav_init(p, x0, start_at_argmin_diag, V, W, ldv, S(stream));
    stream_leave(p, S(stream));
    return rc;
}

static int step_common(Plan *p, double *V, double *W, int64_t ldv, int32_t *k, double *lambda, double *resnorm,
                       int32_t *converged, cudaStream_t st, bool enqueue_only, bool skip_apply = false) {
    if (p->timing.enabled) ensure_timing(p);
    int k_next = *k;
    stream_enter(p, st);
    int rc = dav_enqueue_step(p, V, W, ldv, *k, st, &k_next, skip_apply);
    stream_leave(p, st);
    if (rc != DMRG_OK) return rc;
    if (enqueue_only) {   // no stream synchronisation (see dmrg_davidson_poll)
        *k = k_next;
        return DMRG_OK;
    }
    rc = read_state(p, st, false);
    if (rc != DMRG_OK) return rc;
    const DavState &s = *p->state_host;
    if (lambda) *lambda = s.lambda;
    if (resnorm) *resnorm = s.rho;
    if (converged) *converged = (s.done == 1) ? 1 : 0;
    if (s.error || s.done == 2) return fail(p, DMRG_E_NUMERIC, "Davidson breakdown: zero or non-finite norm");
    if (s.done != 1) *k = k_next;
    if (p->timing.enabled) {
        for (int q = 0; q < 8; q++) {
            float ms = 0.f;
            cudaEventElapsedTime(&ms, p->timing.ev[q], p->timing.ev[q + 1]);
            p->timing.ms[q] = ms;
        }
    }
    return DMRG_OK;
}

int dmrg_davidson_step(dmrg_handle_t h, double *V, double *W, int64_t ldv, int32_t *k, double *lambda,
                       double *resnorm, int32_t *converged, void *stream) {
    if (!h) return DMRG_E_INVALID_ARG;
    Plan *p = P(h);
    if (!V || !W || !k) return fail(p, DMRG_E_INVALID_ARG, "davidson_step: NULL argument");
    return step_common(p, V, W, ldv, k, lambda, resnorm, converged, S(stream), !lambda && !resnorm && !converged);
}

int dmrg_davidson_step_given_w(dmrg_handle_t h, double *V, double *W, int64_t ldv, int32_t *k, double *lambda,
                               double *resnorm, int32_t *converged, void *stream) {
    if (!h) return DMRG_E_INVALID_ARG;
    Plan *p = P(h);
    if (!V || !W || !k) return fail(p, DMRG_E_INVALID_ARG, "davidson_step_given_w: NULL argument");
    return step_common(p, V, W, ldv, k, lambda, resnorm, converged, S(stream), !lambda && !resnorm && !converged, true);
}

int dmrg_partition_outputs(int32_t n_outputs, const int64_t *cost, int32_t n_ranks, int32_t *owner) {
    if (n_outputs < 0 || n_ranks < 1 || !cost || !owner) return fail(nullptr, DMRG_E_INVALID_ARG, "partition_outputs: bad argument");
    std::vector<long long> c(cost, cost + n_outputs);
    partition_outputs(n_outputs, c.data(), n_ranks, owner);
    return DMRG_OK;
}

int dmrg_get_shard(dmrg_handle_t h, int32_t *owner) {
    if (!h || !owner) return DMRG_E_INVALID_ARG;
    Plan *p = P(h);
    for (size_t q = 0; q < p->owner.size(); q++) owner[q] = p->owner[q];
    return DMRG_OK;
}

// Device-accessible alias of a pinned host pointer (cudaHostAlloc / cudaHostRegister memory); NULL for pageable memory.
static void *device_view(const void *host) {
    cudaPointerAttributes a{};
    if (cudaPointerGetAttributes(&a, host) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    return (a.type == cudaMemoryTypeHost) ? a.devicePointer : nullptr;
}

int dmrg_davidson_step_host(dmrg_handle_t h, double *V, double *W, int64_t ldv, int32_t *k, const double *v_in_host,
                            double *w_out_host, double *lambda, double *resnorm, int32_t *converged, void *stream) {
    if (!h) return DMRG_E_INVALID_ARG;
    Plan *p = P(h);
    if (!V || !W || !k) return fail(p, DMRG_E_INVALID_ARG, "davidson_step_host: NULL argument");
    if (*k < 1 || *k > p->opt.k_max || ldv < p->n) return fail(p, DMRG_E_INVALID_ARG, "davidson_step_host: k or ldv out of range");
    cudaStream_t st = S(stream);
    // a run that has already converged makes the step a no-op: do not overwrite a column dmrg_ritz_vector still needs
    if (v_in_host) p->ximg_src = nullptr;       // the newest basis vector comes from the caller: its tile images are not current
    // A pinned (device-accessible) v_in is not copied by the copy engine: loader CTAs of the projection kernel pull it over PCIe
    // share by share while the other CTAs already work on the segments that have arrived (DMRG_HOST_STREAM=0: staged copy).
    // Pageable memory, or a plan with axpy terms (l-1-1-r), takes the staged copy.  (Mirroring H v to the host from the
    // kernel's epilogue was measured too: the scattered 16-byte PCIe writes doubled the step time; w_out stays a D2H copy
    // on the side stream, under lines 3-13.)
    static const int host_stream = []() { const char *e = getenv("DMRG_HOST_STREAM"); return e ? atoi(e) : 1; }();
    const double *v_dev = nullptr;
    if (v_in_host && host_stream && !p->axpy_count) v_dev = static_cast<const double *>(device_view(v_in_host));
    if (v_in_host && p->state_host->done != 1) {
        if (v_dev) p->x_stream = v_dev;
        else cudaMemcpyAsync(V + (long long)(*k - 1) * ldv, v_in_host, sizeof(double) * p->n, cudaMemcpyHostToDevice, st);
    }
    p->w_out_host = w_out_host;
    int rc = step_common(p, V, W, ldv, k, lambda, resnorm, converged, st, false);
    p->w_out_host = nullptr; p->x_stream = nullptr;
    if (w_out_host) {
        cudaError_t e = cudaStreamSynchronize(p->side);
        if (rc == DMRG_OK && e != cudaSuccess) return fail(p, DMRG_E_CUDA, cudaGetErrorString(e));
    }
    return rc;
}

int dmrg_davidson_poll(dmrg_handle_t h, double *lambda, double *resnorm, int32_t *converged, int32_t *iters,
                       void *stream) {
    if (!h) return DMRG_E_INVALID_ARG;
    Plan *p = P(h);
    int rc = read_state(p, S(stream), false);
    if (rc != DMRG_OK) return rc;
    const DavState &st = *p->state_host;
    if (lambda) *lambda = st.lambda;
    if (resnorm) *resnorm = st.rho;
    if (converged) *converged = (st.done == 1) ? 1 : 0;
    if (iters) *iters = st.iters;
    if (st.error || st.done == 2) return fail(p, DMRG_E_NUMERIC, "Davidson breakdown: zero or non-finite norm");
    return DMRG_OK;
}

int dmrg_get_small(dmrg_handle_t h, double *B_host, double *y_host, void *stream) {
    if (!h) return DMRG_E_INVALID_ARG;
    Plan *p = P(h);
    int rc = read_state(p, S(stream));
    if (rc != DMRG_OK) return rc;
    if (B_host) {
        const int km = p->opt.k_max;
        for (int i = 0; i < km; i++) for (int j = 0; j < km; j++) B_host[i * km + j] = p->state_host->B[i * KMAX + j];
    }
    if (y_host) for (int i = 0; i < p->opt.k_max; i++) y_host[i] = p->state_host->y[i];
    return DMRG_OK;
}

int dmrg_set_small(dmrg_handle_t h, const double *B_host, void *stream) {
    if (!h || !B_host) return DMRG_E_INVALID_ARG;
    Plan *p = P(h);
    int rc = read_state(p, S(stream));
    if (rc != DMRG_OK) return rc;
    const int km = p->opt.k_max;
    p->ximg_src = nullptr;      // a resumed state: trust nothing cached about the caller's basis
    memset(p->state_host->B, 0, sizeof(p->state_host->B));
    for (int i = 0; i < km; i++) for (int j = 0; j < km; j++) p->state_host->B[i * KMAX + j] = B_host[i * km + j];
    p->state_host->e_k = 0;   // the kept eigenvectors no longer belong to this B
    cudaError_t e = cudaMemcpyAsync(&p->state->e_k, &p->state_host->e_k, sizeof(int), cudaMemcpyHostToDevice, S(stream));
    if (e == cudaSuccess) e = cudaMemcpyAsync(p->state->B, p->state_host->B, sizeof(p->state_host->B), cudaMemcpyHostToDevice, S(stream));
    if (e == cudaSuccess) e = cudaStreamSynchronize(S(stream));
    return e == cudaSuccess ? DMRG_OK : fail(p, DMRG_E_CUDA, cudaGetErrorString(e));
}

int dmrg_ritz_vector(dmrg_handle_t h, const double *V, int64_t ldv, int32_t k, double *x_out, void *stream) {
    if (!h) return DMRG_E_INVALID_ARG;
    Plan *p = P(h);
    if (!V || !x_out || ldv < p->n) return fail(p, DMRG_E_INVALID_ARG, "ritz_vector: bad argument");
    return dav_ritz(p, V, ldv, k, x_out, S(stream));
}

static int ensure_own_basis(Plan *p) {
    if (p->Vown) return DMRG_OK;
    p->ldv_own = (p->n + 15) / 16 * 16;
    size_t bytes = sizeof(double) * (size_t)p->ldv_own * p->opt.k_max;
    if (cudaMalloc((void **)&p->Vown, bytes) != cudaSuccess || cudaMalloc((void **)&p->Wown, bytes) != cudaSuccess) {
        cudaFree(p->Vown); p->Vown = nullptr; p->Wown = nullptr; cudaGetLastError();
        return fail(p, DMRG_E_ALLOC, "cannot allocate the plan-owned Davidson basis");
    }
    p->device_bytes += 2 * (long long)bytes;
    return DMRG_OK;
}

int dmrg_lowest_eigenpair(dmrg_handle_t h, const double *x0, int32_t start_at_argmin_diag, double *x_out,
                          double *lambda, double *resnorm, int32_t *iters, void *stream) {
    if (!h) return DMRG_E_INVALID_ARG;
    Plan *p = P(h);
    if (!x_out) return fail(p, DMRG_E_INVALID_ARG, "lowest_eigenpair: x_out is NULL");
    cudaStream_t st = S(stream);
    const int k_max = p->opt.k_max;
    { int rcb = ensure_own_basis(p); if (rcb != DMRG_OK) return rcb; }
    const bool was_timing = p->timing.enabled;
    p->timing.enabled = false;
    int rc = dav_init(p, x0, start_at_argmin_diag, p->Vown, p->Wown, p->ldv_own, st);
    int k = 1, done = 0;
    for (int it = 1; rc == DMRG_OK && it <= p->opt.max_iter; it++) {
        int k_next = k;
        rc = dav_enqueue_step(p, p->Vown, p->Wown, p->ldv_own, k, st, &k_next);
        if (rc != DMRG_OK) break;
        k = k_next;
        if (it % p->opt.check_every == 0 || it == p->opt.max_iter) {
            rc = read_state(p, st, false);
            if (rc != DMRG_OK) break;
            done = p->state_host->done;
            if (done) break;
        }
    }
    p->timing.enabled = was_timing;
    if (rc != DMRG_OK) return rc;
    const DavState &s = *p->state_host;
    if (lambda) *lambda = s.lambda;
    if (resnorm) *resnorm = s.rho;
    if (iters) *iters = s.iters;
    if (s.error || done == 2) return fail(p, DMRG_E_NUMERIC, "Davidson breakdown: zero or non-finite norm");
    // Ritz vector of the last executed step; after a restart step V(:,0) already is x/||x||
    if (done != 1 && s.k_used == k_max)
        cudaMemcpyAsync(x_out, p->Vown, sizeof(double) * p->n, cudaMemcpyDeviceToDevice, st);
    else
        rc = dav_ritz(p, p->Vown, p->ldv_own, s.k_used, x_out, st);
    if (rc != DMRG_OK) return rc;
    cudaError_t e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return fail(p, DMRG_E_CUDA, cudaGetErrorString(e));
    return done == 1 ? DMRG_OK : DMRG_NOT_CONVERGED;
}

int dmrg_apply_H_multi(dmrg_handle_t h, int32_t nrhs, const double *x, int64_t ldx, double *y, int64_t ldy, void *stream) {
    if (!h) return DMRG_E_INVALID_ARG;
    Plan *p = P(h);
    if (!x || !y || ldx < p->n || ldy < p->n) return fail(p, DMRG_E_INVALID_ARG, "apply_H_multi: NULL vectors or a column stride below n");
    const double *xe = x + (nrhs - 1) * ldx + p->n; const double *ye = y + (nrhs - 1) * ldy + p->n;
    if (!(xe <= y || ye <= x)) return fail(p, DMRG_E_INVALID_ARG, "apply_H_multi: x and y overlap");
    stream_enter(p, S(stream));
    const int rc = apply_H(p, x, y, nullptr, S(stream), nullptr, nrhs, ldx, ldy);
    stream_leave(p, S(stream));
    return rc;
}

int dmrg_block_init(dmrg_handle_t h, int32_t nb, const double *X0, int64_t ldx0, double *V, double *W, int64_t ldv, void *stream) {
    if (!h) return DMRG_E_INVALID_ARG;
    return bdav_init(P(h), nb, X0, ldx0, V, W, ldv, S(stream));
}

int dmrg_block_step(dmrg_handle_t h, double *V, double *W, int64_t ldv, int32_t *k, int32_t *na, int32_t nb, double *theta,
                    double *resnorm, int32_t *converged, void *stream) {
    if (!h) return DMRG_E_INVALID_ARG;
    Plan *p = P(h);
    if (!V || !W || !k || !na) return fail(p, DMRG_E_INVALID_ARG, "block_step: NULL argument");
    int kk = *k, nn = *na;
    stream_enter(p, S(stream));
    int rc = bdav_step(p, V, W, ldv, &kk, &nn, nb, theta, resnorm, converged, S(stream));
    stream_leave(p, S(stream));
    if (rc == DMRG_OK) { *k = kk; *na = nn; }
    return rc;
}

int dmrg_block_ritz(dmrg_handle_t h, const double *V, const double *W, int64_t ldv, int32_t k, int32_t nb, double *X_out,
                    int64_t ldxo, void *stream) {
    if (!h) return DMRG_E_INVALID_ARG;
    if (!V || !W || !X_out) return fail(P(h), DMRG_E_INVALID_ARG, "block_ritz: NULL argument");
    return bdav_ritz(P(h), V, W, ldv, k, nb, X_out, ldxo, S(stream));
}

int dmrg_block_get_small(dmrg_handle_t h, int32_t nb, double *G_host, double *Y_host, void *stream) {
    if (!h) return DMRG_E_INVALID_ARG;
    Plan *p = P(h);
    if (!p->bstate || nb < 1 || nb > BMAX) return fail(p, DMRG_E_INVALID_ARG, "block_get_small: no block state (options.max_rhs) or bad nb");
    cudaError_t e = cudaMemcpyAsync(p->bstate_host, p->bstate, sizeof(BlockState), cudaMemcpyDeviceToHost, S(stream));
    if (e == cudaSuccess) e = cudaStreamSynchronize(S(stream));
    if (e != cudaSuccess) return fail(p, DMRG_E_CUDA, cudaGetErrorString(e));
    const int km = p->opt.k_max;
    if (G_host) for (int i = 0; i < km; i++) for (int j = 0; j < km; j++) G_host[i * km + j] = p->bstate_host->G[i * KMAX + j];
    if (Y_host) for (int i = 0; i < km; i++) for (int r = 0; r < nb; r++) Y_host[i * nb + r] = p->bstate_host->Y[i * BMAX + r];
    return DMRG_OK;
}

int dmrg_block_lowest_eigenpairs(dmrg_handle_t h, int32_t nb, const double *X0, int64_t ldx0, double *X_out, int64_t ldxo,
                                 double *theta, double *resnorm, int32_t *iters, int32_t *applies, void *stream) {
    if (!h) return DMRG_E_INVALID_ARG;
    Plan *p = P(h);
    if (!X_out) return fail(p, DMRG_E_INVALID_ARG, "block_lowest_eigenpairs: X_out is NULL");
    int rc = ensure_own_basis(p);
    if (rc != DMRG_OK) return rc;
    cudaStream_t st = S(stream);
    rc = bdav_init(p, nb, X0, ldx0, p->Vown, p->Wown, p->ldv_own, st);
    int k = nb, na = nb, it = 0, ap = 0, conv = 0, k_used = nb;
    while (rc == DMRG_OK && ap < p->opt.max_iter) {
        it++; ap += na; k_used = k;
        rc = bdav_step(p, p->Vown, p->Wown, p->ldv_own, &k, &na, nb, theta, resnorm, &conv, st);
        if (conv) break;
    }
    if (iters) *iters = it;
    if (applies) *applies = ap;
    if (rc != DMRG_OK) return rc;
    rc = bdav_ritz(p, p->Vown, p->Wown, p->ldv_own, k_used, nb, X_out, ldxo, st);
    if (rc != DMRG_OK) return rc;
    cudaError_t e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return fail(p, DMRG_E_CUDA, cudaGetErrorString(e));
    return conv ? DMRG_OK : DMRG_NOT_CONVERGED;
}

int dmrg_gemv_trans(dmrg_handle_t h, const double *V, int64_t ldv, int32_t k, const double *w, double *out, void *stream) {
    if (!h || !V || !w || !out) return DMRG_E_INVALID_ARG;
    return dav_gemv_trans(P(h), V, ldv, k, w, out, S(stream));
}

int dmrg_gemv_trans_static(const double *V, int64_t ldv, int64_t n, int32_t k, const double *w, double *out, void *stream) {
    return dav_gemv_trans_static(V, ldv, n, k, w, out, S(stream));
}

int dmrg_gemv_sub(dmrg_handle_t h, const double *V, int64_t ldv, int32_t k, const double *s, double *t,
                  double *nrm2_out, void *stream) {
    if (!h || !V || !s || !t || !nrm2_out) return DMRG_E_INVALID_ARG;
    return dav_gemv_sub(P(h), V, ldv, k, s, t, nrm2_out, S(stream));
}

int dmrg_probe_fp64_peak(int32_t kind, int32_t reps, double *tflops, void *stream) {
    if (!tflops || reps < 1 || kind < 0 || kind > 1) return DMRG_E_INVALID_ARG;
    return probe_fp64(kind, reps, tflops, S(stream));
}

int dmrg_probe_hbm_read(int64_t bytes, int32_t reps, double *gbs, void *stream) {
    if (!gbs || reps < 1) return DMRG_E_INVALID_ARG;
    return probe_hbm(bytes, reps, gbs, S(stream));
}

int dmrg_get_unit_trace(dmrg_handle_t h, uint64_t *trace_host, int32_t max_units, int32_t *n_units) {
    if (!h || !n_units) return DMRG_E_INVALID_ARG;
    Plan *p = P(h);
    *n_units = 0;
    if (!p->trace || !trace_host || max_units <= 0) return DMRG_OK;
    const int nu = p->trace_units < max_units ? p->trace_units : max_units;
    cudaError_t e = cudaDeviceSynchronize();
    if (e == cudaSuccess) e = cudaMemcpy(trace_host, p->trace, 32 * (size_t)nu, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return fail(p, DMRG_E_CUDA, cudaGetErrorString(e));
    *n_units = nu;
    return DMRG_OK;
}

int dmrg_set_timing(dmrg_handle_t h, int32_t enable) {
    if (!h) return DMRG_E_INVALID_ARG;
    P(h)->timing.enabled = enable != 0;
    if (enable) ensure_timing(P(h));
    return DMRG_OK;
}

int dmrg_get_timing(dmrg_handle_t h, double *ms8) {
    if (!h || !ms8) return DMRG_E_INVALID_ARG;
    for (int q = 0; q < 8; q++) ms8[q] = P(h)->timing.ms[q];
    return DMRG_OK;
}

}  // extern "C"
