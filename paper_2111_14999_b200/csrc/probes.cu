// probes.cu -- measurement aids, built into their OWN shared library (libphoebe_elph_probes.so, include/
// phoebe_elph_probes.h): FP64 and HBM ceiling probes for the roofline denominators of bench.py.  Not part of the product
// library: libphoebe_elph.so exports only the calls of the hot path.
#include "../../include/phoebe_elph_probes.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cstdint>

#include "probe_kernels.cuh"

namespace {
constexpr int kSMs = 148;
constexpr int PHOEBE_ELPH_OK = 0, PHOEBE_ELPH_E_NULL = -1, PHOEBE_ELPH_E_DIMS = -2, PHOEBE_ELPH_E_CUDA = -6;
bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
}  // namespace

extern "C" {

int phoebe_elph_probe_fp64(int32_t kind, int32_t iters, void* cuda_stream, double* tflops_out)
{
    if (!tflops_out) return PHOEBE_ELPH_E_NULL;
    if (kind < 0 || kind > 1 || iters <= 0) return PHOEBE_ELPH_E_DIMS;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const int grid = kSMs * 4, threads = 256;
    double* out = nullptr;
    if (cudaMalloc(&out, (size_t)grid * threads * 8) != cudaSuccess) return PHOEBE_ELPH_E_CUDA;
    cudaEvent_t a, b;
    cudaEventCreate(&a); cudaEventCreate(&b);
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(a, st);
        if (kind == 0) pe::k_probe_dfma<<<grid, threads, 0, st>>>(out, iters, 1.0000001, 1e-9);
        else pe::k_probe_dmma<<<grid, threads, 0, st>>>(out, iters, 1.0000001, 1e-9);
        cudaEventRecord(b, st);
        if (cudaEventSynchronize(b) != cudaSuccess) { cudaFree(out); return PHOEBE_ELPH_E_CUDA; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, a, b);
        if (rep > 0) best = std::min(best, ms);
    }
    cudaEventDestroy(a); cudaEventDestroy(b);
    cudaFree(out);
    const double fma_per_thread_iter = (kind == 0) ? 64.0 : (32.0 * 256.0 / 32.0);   // DMMA: 256 FMA per warp instr
    const double flops = 2.0 * fma_per_thread_iter * iters * (double)grid * threads;
    *tflops_out = flops / (best * 1e-3) * 1e-12;
    return PHOEBE_ELPH_OK;
}

int phoebe_elph_probe_hbm_read(const void* buf_dev, size_t bytes, void* cuda_stream, double* gbs_out)
{
    if (!buf_dev || !gbs_out) return PHOEBE_ELPH_E_NULL;
    if (bytes < 16 || !aligned16(buf_dev)) return PHOEBE_ELPH_E_DIMS;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    double* out = nullptr;
    if (cudaMalloc(&out, 8) != cudaSuccess) return PHOEBE_ELPH_E_CUDA;
    cudaEvent_t a, b;
    cudaEventCreate(&a); cudaEventCreate(&b);
    float best = 1e30f;
    for (int rep = 0; rep < 6; ++rep) {
        cudaEventRecord(a, st);
        pe::k_probe_read<<<kSMs * 8, 256, 0, st>>>(static_cast<const double2*>(buf_dev), bytes / 16, out);
        cudaEventRecord(b, st);
        if (cudaEventSynchronize(b) != cudaSuccess) { cudaFree(out); return PHOEBE_ELPH_E_CUDA; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, a, b);
        if (rep > 0) best = std::min(best, ms);
    }
    cudaEventDestroy(a); cudaEventDestroy(b);
    cudaFree(out);
    *gbs_out = (double)(bytes / 16 * 16) / (best * 1e-3) * 1e-9;
    return PHOEBE_ELPH_OK;
}

}  // extern "C"
