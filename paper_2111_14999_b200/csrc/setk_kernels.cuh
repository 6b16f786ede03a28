// setk_kernels.cuh -- steps a1 + a2 (Eq. 71): the fixed-k precompute.
//
//   a1  T[p][x]        = sum_e (e^{2 pi i k.Re_e}/deg_e[e]) g_W[p][e][x]      x = (w1,w2,kappa) flattened
//   a2  g1[p][b1][y]   = sum_{w1} U_k[w1][b1] T[p][w1][y]                      y = (w2,kappa) flattened
//
// a1 streams g_W exactly once (0.5 flop/B: HBM-bound).  Work item = (p, Re-chunk s,
// tile of x): fully coalesced 128-bit loads, >= UE independent loads in flight per
// thread, many small items so the tail never starves HBM.  Partial sums over the
// Re-chunks go to Tpart[s][p][x]; a2 adds them in fixed order (deterministic) and
// rotates in registers.
#pragma once
#include "ptx_helpers.cuh"

namespace pe {

constexpr int SETK_UE = 8;   // e-unroll = independent 16-B loads in flight per thread

__global__ void __launch_bounds__(256)
k_setk_stream(const double2* __restrict__ gW, const double* __restrict__ Re, const double* __restrict__ deg_e,
              double k0, double k1, double k2, int nRe, int nRp, int X, int epc,
              double2* __restrict__ Tpart /* [S][nRp][X] */)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double2* ph = reinterpret_cast<double2*>(smem_raw);          // [epc]
    const int p = blockIdx.z, s = blockIdx.y;
    const int e0 = s * epc;
    const int ne = min(epc, nRe - e0);
    // phases of this Re-chunk (a few hundred sincospi per CTA, negligible vs the stream)
    for (int i = threadIdx.x; i < ne; i += blockDim.x) {
        const double* R = Re + 3 * (size_t)(e0 + i);
        double x = k0 * R[0] + k1 * R[1] + k2 * R[2];
        double sn, cs;
        sincospi(2.0 * x, &sn, &cs);
        double w = 1.0 / deg_e[e0 + i];
        ph[i] = make_double2(cs * w, sn * w);
    }
    __syncthreads();
    const int col = blockIdx.x * blockDim.x + threadIdx.x;
    if (col >= X) return;
    const double2* g = gW + ((size_t)p * nRe + e0) * (size_t)X + col;
    double ar = 0.0, ai = 0.0;
    int e = 0;
    for (; e + SETK_UE <= ne; e += SETK_UE) {
        double2 v[SETK_UE];
#pragma unroll
        for (int u = 0; u < SETK_UE; ++u) v[u] = ld_stream(g + (size_t)(e + u) * X);
#pragma unroll
        for (int u = 0; u < SETK_UE; ++u) {
            const double2 f = ph[e + u];
            ar = fma(f.x, v[u].x, ar); ar = fma(-f.y, v[u].y, ar);
            ai = fma(f.x, v[u].y, ai); ai = fma(f.y, v[u].x, ai);
        }
    }
    for (; e < ne; ++e) {
        const double2 v = ld_stream(g + (size_t)e * X);
        const double2 f = ph[e];
        ar = fma(f.x, v.x, ar); ar = fma(-f.y, v.y, ar);
        ai = fma(f.x, v.y, ai); ai = fma(f.y, v.x, ai);
    }
    Tpart[((size_t)s * nRp + p) * (size_t)X + col] = make_double2(ar, ai);
}

// a2: one thread per (p, y), NBT values of b1 per thread.  blockIdx.z = ik * ngroups + (b1 group):
// a batch of k-points (set_k_batch) is rotated by one launch; k-point ik reads Tpart + ik*strideT,
// Uk + ik*nw*nb1 and writes g1 + ik*strideG.
template <int NBT>
__global__ void __launch_bounds__(128)
k_setk_rotate(const double2* __restrict__ Tpart, const double2* __restrict__ Uk /* [nk][nw][nb1] */,
              int S, int nRp, int nw, int Y, int nb1, double2* __restrict__ g1 /* [nk][nRp][nb1][Y] */, int ldg,
              int ngroups, long long strideT, long long strideG, int conjU /* set_conventions: U_k enters conjugated */)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double2* U = reinterpret_cast<double2*>(smem_raw);           // [nw][NBT]
    const int ik = blockIdx.z / ngroups;
    const int b0 = (blockIdx.z - ik * ngroups) * NBT;
    Tpart += (size_t)ik * strideT;
    Uk += (size_t)ik * nw * nb1;
    g1 += (size_t)ik * strideG;
    for (int i = threadIdx.x; i < nw * NBT; i += blockDim.x) {
        int w1 = i / NBT, b = i % NBT;
        double2 u = (b0 + b < nb1) ? Uk[(size_t)w1 * nb1 + b0 + b] : make_double2(0.0, 0.0);
        if (conjU) u.y = -u.y;
        U[i] = u;
    }
    __syncthreads();
    const int p = blockIdx.y;
    const int y = blockIdx.x * blockDim.x + threadIdx.x;
    if (y >= Y) return;
    const size_t X = (size_t)nw * Y;
    double ar[NBT], ai[NBT];
#pragma unroll
    for (int b = 0; b < NBT; ++b) { ar[b] = 0.0; ai[b] = 0.0; }
    for (int w1 = 0; w1 < nw; ++w1) {
        double tr = 0.0, ti = 0.0;
        for (int s = 0; s < S; ++s) {
            const double2 t = Tpart[((size_t)s * nRp + p) * X + (size_t)w1 * Y + y];
            tr += t.x; ti += t.y;
        }
#pragma unroll
        for (int b = 0; b < NBT; ++b) {
            const double2 u = U[w1 * NBT + b];
            ar[b] = fma(u.x, tr, ar[b]); ar[b] = fma(-u.y, ti, ar[b]);
            ai[b] = fma(u.x, ti, ai[b]); ai[b] = fma(u.y, tr, ai[b]);
        }
    }
#pragma unroll
    for (int b = 0; b < NBT; ++b)
        if (b0 + b < nb1) g1[(size_t)p * ldg + (size_t)(b0 + b) * Y + y] = make_double2(ar[b], ai[b]);
}

}  // namespace pe
