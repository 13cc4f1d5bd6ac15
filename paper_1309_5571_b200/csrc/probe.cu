// probe.cu -- register-only issue-rate probes: the FP64 roofline denominator measured on the box
// (MEASURED_PEAKS.json carries no FP64 entry) and a read-only HBM stream.
#include "internal.h"

namespace dmrg {
namespace {

__global__ void dfma_probe_kernel(double *out, int iters, double a, double b) {
    double acc[16];
#pragma unroll
    for (int i = 0; i < 16; i++) acc[i] = threadIdx.x * 1e-3 + i;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 16; i++) acc[i] = fma(acc[i], a, b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 16; i++) s += acc[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void dmma_probe_kernel(double *out, int iters, double a, double b) {
    double c[16][2];
#pragma unroll
    for (int i = 0; i < 16; i++) { c[i][0] = threadIdx.x * 1e-3 + i; c[i][1] = i; }
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 16; i++)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                         : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 16; i++) s += c[i][0] + c[i][1];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void read_probe_kernel(const double2 *__restrict__ p, size_t n2, double *out) {
    size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x, stride = (size_t)gridDim.x * blockDim.x;
    double s = 0;
    for (; i + 3 * stride < n2; i += 4 * stride) {
        double2 a = p[i], b = p[i + stride], c = p[i + 2 * stride], d = p[i + 3 * stride];
        s += a.x + a.y + b.x + b.y + c.x + c.y + d.x + d.y;
    }
    for (; i < n2; i += stride) { double2 a = p[i]; s += a.x + a.y; }
    if (s == 1.2345e300) out[0] = s;
}

}  // namespace

int probe_fp64(int kind, int reps, double *tflops, cudaStream_t st) {
    int dev = 0, nsm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return fail(nullptr, DMRG_E_CUDA, "no CUDA device");
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    const int threads = 512, blocks = nsm, iters = (kind == 0) ? 40000 : 10000;
    double *out = nullptr;
    if (cudaMalloc(&out, sizeof(double) * threads * blocks) != cudaSuccess) return fail(nullptr, DMRG_E_ALLOC, "probe alloc");
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    double best = 0.0;
    for (int r = 0; r < reps + 1; r++) {
        cudaEventRecord(e0, st);
        if (kind == 0) dfma_probe_kernel<<<blocks, threads, 0, st>>>(out, iters, 1.0000001, 1e-9);
        else dmma_probe_kernel<<<blocks, threads, 0, st>>>(out, iters, 1.0000001, 1e-9);
        cudaEventRecord(e1, st);
        cudaEventSynchronize(e1);
        float ms = 0; cudaEventElapsedTime(&ms, e0, e1);
        const double fl = (kind == 0) ? 2.0 * 16 * iters * (double)threads * blocks
                                      : 2.0 * 256 * 16 * iters * (double)(threads / 32) * blocks;
        if (r > 0 && ms > 0) best = fmax(best, fl / ms / 1e9);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(out);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(nullptr, DMRG_E_CUDA, cudaGetErrorString(e));
    *tflops = best;
    return DMRG_OK;
}

int probe_hbm(long long bytes, int reps, double *gbs, cudaStream_t st) {
    int dev = 0, nsm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return fail(nullptr, DMRG_E_CUDA, "no CUDA device");
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    double2 *buf = nullptr; double *out = nullptr;
    bytes = (bytes / 16) * 16;
    if (bytes <= 0) return fail(nullptr, DMRG_E_INVALID_ARG, "probe_hbm: bytes");
    if (cudaMalloc(&buf, bytes) != cudaSuccess || cudaMalloc(&out, 8) != cudaSuccess) { cudaFree(buf); return fail(nullptr, DMRG_E_ALLOC, "probe alloc"); }
    cudaMemsetAsync(buf, 0, bytes, st);
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    double best = 0.0;
    for (int r = 0; r < reps + 1; r++) {
        cudaEventRecord(e0, st);
        read_probe_kernel<<<nsm * 16, 256, 0, st>>>(buf, (size_t)bytes / 16, out);
        cudaEventRecord(e1, st);
        cudaEventSynchronize(e1);
        float ms = 0; cudaEventElapsedTime(&ms, e0, e1);
        if (r > 0 && ms > 0) best = fmax(best, (double)bytes / ms / 1e6);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(buf); cudaFree(out);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(nullptr, DMRG_E_CUDA, cudaGetErrorString(e));
    *gbs = best;
    return DMRG_OK;
}

}  // namespace dmrg
