// noalloc.cu -- phoebe_elph_set_k_noalloc: steps a1 + a2 (Eq. 71) for callers that cannot allocate
// (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).  The context-based path keeps the Fourier-summed,
// not yet rotated tensor T[p][w1][w2][kappa] in the caller's workspace; this variant keeps it in a FILE-SCOPE device array
// of fixed size, so that the call needs no workspace, no context and no allocation of any kind.
//
//   a1  T[p][x]      = sum_e (e^{2 pi i k.Re_e} / deg_e[e]) g_W[p][e][x]        x = (w1, w2, kappa)      -> scratch
//   a2  g1'[p][b1][y] = sum_{w1} U_k[w1][b1] T[p][w1][y]                          y = (w2, kappa)          -> caller's output
//
// The array exists once per GPU that loads the library (PHOEBE_ELPH_NOALLOC_MAX_BYTES, held until the process exits) and
// is SHARED by every call: it keeps the last call's contents (every element a call reads it has written first, so nothing
// needs clearing), and two calls that overlap on the GPU (different streams, or graphs replayed concurrently) RACE.
#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <mutex>

#include "../../include/phoebe_elph.h"

namespace {

constexpr size_t kScratchElems = PHOEBE_ELPH_NOALLOC_MAX_BYTES / sizeof(double2);
static __device__ __align__(256) double2 g_noalloc_scratch[kScratchElems];

// In host code `g_noalloc_scratch` is only a handle of the symbol, not a device address: the address is looked up once per
// device (cudaGetSymbolAddress, with that device current) and passed to the kernels as an ordinary pointer.
constexpr int kMaxDevices = 64;
double2* g_scratch_addr[kMaxDevices] = {};
std::mutex g_mu;
thread_local char g_err[256] = "";

int fail(int code, const char* fmt, const char* detail = "")
{
    std::snprintf(g_err, sizeof(g_err), fmt, detail);
    return code;
}

int scratch_for_current_device(double2** out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(PHOEBE_ELPH_E_CUDA, "noalloc: cudaGetDevice: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= kMaxDevices) return fail(PHOEBE_ELPH_E_DIMS, "noalloc: device ordinal beyond %s", "63");
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_addr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess || !p) return fail(PHOEBE_ELPH_E_CUDA, "noalloc: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
        g_scratch_addr[dev] = static_cast<double2*>(p);
    }
    *out = g_scratch_addr[dev];
    return PHOEBE_ELPH_OK;
}

constexpr int kPhaseChunk = 512;      // Re vectors whose phases are staged in shared memory at a time (8 KB)

// a1: one thread per (p, x); the Re sum runs in list order (deterministic).  grid (ceil(X / 128), nRp), block 128.
__global__ void __launch_bounds__(128)
k_na_fourier(const double2* __restrict__ gW, const double* __restrict__ Re, const double* __restrict__ deg_e, double k0,
             double k1, double k2, int nRe, int X, double2* __restrict__ T /* [nRp][X] */)
{
    __shared__ double2 ph[kPhaseChunk];
    const int p = blockIdx.y, x = blockIdx.x * 128 + threadIdx.x;
    const double2* g = gW + (size_t)p * nRe * (size_t)X + x;
    double ar = 0.0, ai = 0.0;
    for (int e0 = 0; e0 < nRe; e0 += kPhaseChunk) {
        const int ne = min(kPhaseChunk, nRe - e0);
        __syncthreads();
        for (int i = threadIdx.x; i < ne; i += 128) {
            const double* R = Re + 3 * (size_t)(e0 + i);
            double sn, cs;
            sincospi(2.0 * (k0 * R[0] + k1 * R[1] + k2 * R[2]), &sn, &cs);
            const double w = deg_e ? 1.0 / deg_e[e0 + i] : 1.0;
            ph[i] = make_double2(cs * w, sn * w);
        }
        __syncthreads();
        if (x < X) {
#pragma unroll 4
            for (int e = 0; e < ne; ++e) {
                const double2 v = g[(size_t)(e0 + e) * X];
                const double2 f = ph[e];
                ar = fma(f.x, v.x, ar); ar = fma(-f.y, v.y, ar);
                ai = fma(f.x, v.y, ai); ai = fma(f.y, v.x, ai);
            }
        }
    }
    if (x < X) T[(size_t)p * X + x] = make_double2(ar, ai);
}

// a2: one thread per (p, b1, y).  grid (ceil(Y / 128), nb1, nRp), block 128.
__global__ void __launch_bounds__(128)
k_na_rotate(const double2* __restrict__ T, const double2* __restrict__ Uk /* [nw][nb1] */, int nw, int Y, int nb1,
            double2* __restrict__ g1 /* [nRp][nb1][Y] */)
{
    const int y = blockIdx.x * 128 + threadIdx.x, b1 = blockIdx.y, p = blockIdx.z;
    if (y >= Y) return;
    const double2* t = T + (size_t)p * nw * (size_t)Y + y;
    double ar = 0.0, ai = 0.0;
    for (int w1 = 0; w1 < nw; ++w1) {
        const double2 u = Uk[(size_t)w1 * nb1 + b1], v = t[(size_t)w1 * Y];
        ar = fma(u.x, v.x, ar); ar = fma(-u.y, v.y, ar);
        ai = fma(u.x, v.y, ai); ai = fma(u.y, v.x, ai);
    }
    g1[((size_t)p * nb1 + b1) * (size_t)Y + y] = make_double2(ar, ai);
}

}  // namespace

extern "C" {

int phoebe_elph_noalloc_setup(void)
{
    double2* p = nullptr;
    return scratch_for_current_device(&p);
}

int phoebe_elph_set_k_noalloc(const void* gW_dev, const double* Re_dev, const double* deg_e_dev, int32_t nRe, int32_t nRp,
                              int32_t nw, int32_t nmodes, int32_t nb1, const double* k_host, const void* Uk_dev,
                              void* g1_out_dev, void* cuda_stream)
{
    if (!gW_dev || !Re_dev || !k_host || !Uk_dev || !g1_out_dev) return fail(PHOEBE_ELPH_E_NULL, "set_k_noalloc: NULL %s", "pointer");
    if (nRe <= 0 || nRp <= 0 || nw <= 0 || nmodes <= 0 || nb1 <= 0 || nb1 > nw)
        return fail(PHOEBE_ELPH_E_DIMS, "set_k_noalloc: dimensions must be positive and nb1 <= %s", "nw");
    if ((reinterpret_cast<uintptr_t>(gW_dev) | reinterpret_cast<uintptr_t>(Uk_dev) | reinterpret_cast<uintptr_t>(g1_out_dev)) & 15)
        return fail(PHOEBE_ELPH_E_ALIGN, "set_k_noalloc: complex pointers must be 16-byte %s", "aligned");
    const size_t X = (size_t)nw * nw * nmodes, need = (size_t)nRp * X;
    if (need > kScratchElems || nRp > 65535 || nb1 > 65535) {
        std::snprintf(g_err, sizeof(g_err),
                      "set_k_noalloc: nRp * nw * nw * nmodes = %zu complex values exceed the fixed scratch of %zu "
                      "(PHOEBE_ELPH_NOALLOC_MAX_BYTES = %zu bytes); use phoebe_elph_set_k with a workspace",
                      need, kScratchElems, (size_t)PHOEBE_ELPH_NOALLOC_MAX_BYTES);
        return PHOEBE_ELPH_E_DIMS;
    }
    double2* T = nullptr;
    if (int rc = scratch_for_current_device(&T)) return rc;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const int Y = nw * nmodes;
    k_na_fourier<<<dim3((unsigned)((X + 127) / 128), nRp), 128, 0, stream>>>(static_cast<const double2*>(gW_dev), Re_dev, deg_e_dev,
                                                                            k_host[0], k_host[1], k_host[2], nRe, (int)X, T);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(PHOEBE_ELPH_E_CUDA, "set_k_noalloc: k_na_fourier: %s", cudaGetErrorString(e));
    k_na_rotate<<<dim3((Y + 127) / 128, nb1, nRp), 128, 0, stream>>>(T, static_cast<const double2*>(Uk_dev), nw, Y, nb1,
                                                                    static_cast<double2*>(g1_out_dev));
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(PHOEBE_ELPH_E_CUDA, "set_k_noalloc: k_na_rotate: %s", cudaGetErrorString(e));
    return PHOEBE_ELPH_OK;
}

const char* phoebe_elph_noalloc_last_error(void) { return g_err; }

}  // extern "C"
