// setk_pair.cuh -- step a1 for a batch of k-points (Eq. 71) with the +R / -R pairs of the
// ELECTRON lattice vectors folded, as contract_pair.cuh does for the phonon ones:
//     w e^{i th} a + w e^{-i th} b = (w cos th)(a + b) + (w sin th)(i (a - b)),   a = g_W[p][e][x], b = g_W[p][ebar][x]
// so T[k][p][x] = sum_e (e^{2 pi i k.Re}/deg_e) g_W[p][e][x] is a REAL x complex GEMM per phonon vector p: 2 DMMA per tile
// and k-step instead of 3 (three-multiply product).  g_W is borrowed as stored, so the sums a +- b are formed on the
// fly: the producer brings the two rows of a pair into adjacent rows of a ring stage (a bulk copy each, any row order),
// and a lane of the consumer loads both and forms ITS row of the B fragment -- the cosine row (a + b) for even k, the
// sine row i (a - b) for odd k (2 LDS.128 + 2 DFMA per fragment instead of 1 + 1).  At 16 k-points the 4-atom launch
// goes from FP64-bound (85 % of the DMMA peak) to HBM-bound.
//   Ptk  [KrPad][32]       real phases, row 2j = w cos th_j, row 2j+1 = w sin th_j of pair j, k-point contiguous
//   rowmap [Kr]            g_W row (index e) behind ring row r: rowmap[2j] = e, rowmap[2j+1] = ebar, or -1: the zero row
//   zero [X]               a row of zeros (partner-less and self-inverse vectors)
// One tile (all k-points x BN columns of one p) per CTA, as the three-multiply form of this GEMM (k_contract): the
// next CTA's prologue keeps loads in flight while this one stores.
#pragma once
#include "ptx_helpers.cuh"

namespace pe {

template <int BM, int BN, int WN, int KC, int ST>
struct SetkPairCfg {
    static constexpr int kConsumerWarps = WN;
    static constexpr int kThreads = (WN + 1) * 32;
    static constexpr int TM = BM / 8, TN = BN / WN / 8;
    static constexpr int LDA = BM + 4;      // doubles per shared A row (= 32 B mod 128 B for BM = 8, 16, 32)
    static constexpr int LDB = BN + 2;      // complex per shared B row
    static constexpr size_t kRingBytes = (size_t)ST * KC * ((size_t)LDA * 8 + (size_t)LDB * 16);
    static constexpr size_t kSmemBytes = kRingBytes + 2 * ST * sizeof(uint64_t);
    static_assert(KC % 4 == 0 && KC <= 32 && BM % 8 == 0 && BN % (WN * 8) == 0, "tile shape");
};

// A rows for a batch of k-points: Ptk[2j][ik] = w_j cos(2 pi k.R_j), Ptk[2j+1][ik] = sgn w_j sin(2 pi k.R_j); zero for
// ik >= nk and rows >= 2 npairs.  grid (1, rows), block 32 (nk <= 32).
__global__ void __launch_bounds__(32)
k_kphase_pair(const double* __restrict__ k /* [nk][3] */, const double* __restrict__ Rpair /* [npairs][3] */,
              const double* __restrict__ wpair, int nk, int npairs, int KrPad, double sgn, double* __restrict__ Ptk)
{
    const int ik = threadIdx.x;
    for (int j = blockIdx.y; 2 * j < KrPad; j += gridDim.y) {
        double vc = 0.0, vs = 0.0;
        if (ik < nk && j < npairs) {
            const double x = k[3 * ik] * Rpair[3 * j] + k[3 * ik + 1] * Rpair[3 * j + 1] + k[3 * ik + 2] * Rpair[3 * j + 2];
            double sn, cs;
            sincospi(2.0 * x, &sn, &cs);
            vc = wpair[j] * cs; vs = wpair[j] * sgn * sn;
        }
        Ptk[(size_t)(2 * j) * 32 + ik] = vc;
        if (2 * j + 1 < KrPad) Ptk[(size_t)(2 * j + 1) * 32 + ik] = vs;
    }
}

// T[k][p][x] (ldc = nRp X, per-p offset X); M = nk <= BM, N = X, K = 2 npairs, Kpad a multiple of KC.
template <int BM, int BN, int WN, int KC, int ST>
__global__ void __launch_bounds__((WN + 1) * 32, 2)
k_setk_pair(const double* __restrict__ Ptk, const double2* __restrict__ gW, long long strideP /* nRe X */, int X,
            const int* __restrict__ rowmap, const double2* __restrict__ zero, double2* __restrict__ T, long long ldc,
            int M, int K, int Kpad, int nRp)
{
    using Cfg = SetkPairCfg<BM, BN, WN, KC, ST>;
    constexpr int TM = Cfg::TM, TN = Cfg::TN, LDA = Cfg::LDA, LDB = Cfg::LDB, KS = KC / 4;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* As = reinterpret_cast<double*>(smem_raw);                          // [ST][KC][LDA]
    double2* Bs = reinterpret_cast<double2*>(As + (size_t)ST * KC * LDA);      // [ST][KC][LDB]
    uint64_t* full = reinterpret_cast<uint64_t*>(Bs + (size_t)ST * KC * LDB);
    uint64_t* empty = full + ST;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int i = threadIdx.x; i < (int)(Cfg::kRingBytes / 16); i += Cfg::kThreads)
        reinterpret_cast<double2*>(smem_raw)[i] = make_double2(0.0, 0.0);
    if (threadIdx.x == 0) {
        for (int s = 0; s < ST; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, Cfg::kConsumerWarps); }
        mbar_fence_init();
    }
    fence_proxy_async();
    __syncthreads();
    const int ntn = (X + BN - 1) / BN;
    const int p = blockIdx.x / ntn, tn = blockIdx.x - p * ntn;
    const int n0 = tn * BN, bn = min(BN, X - n0);
    const int nchunks = Kpad / KC;
    (void)nRp;

    if (warp == WN) {
        // ---------------- producer warp: one bulk copy per operand row ----------------
        const double2* gp = gW + (size_t)p * strideP + n0;
        int s = 0; uint32_t ph = 0;
        for (int c = 0; c < nchunks; ++c) {
            mbar_wait(empty + s, ph ^ 1u);
            const int k0 = c * KC;
            const int rows_b = max(0, min(KC, K - k0));
            if (lane == 0) mbar_arrive_expect_tx(full + s, (uint32_t)(KC * BM * 8 + rows_b * bn * 16));
            __syncwarp();
            if (lane < KC)
                bulk_g2s(As + ((size_t)s * KC + lane) * LDA, Ptk + (size_t)(k0 + lane) * 32, BM * 8, full + s);
            if (lane < rows_b) {
                const int e = rowmap[k0 + lane];
                const double2* src = e >= 0 ? gp + (size_t)e * X : zero + n0;
                bulk_g2s(Bs + ((size_t)s * KC + lane) * LDB, src, (uint32_t)bn * 16u, full + s);
            }
            if (++s == ST) { s = 0; ph ^= 1u; }
        }
        return;
    }

    // ---------------- consumer warps ----------------
    const int g = lane >> 2, t = lane & 3;
    const double sig = (t & 1) ? -1.0 : 1.0;                 // even k rows: a + b; odd: i (a - b)
    double cr[TM][TN][2], ci[TM][TN][2];
#pragma unroll
    for (int i = 0; i < TM; ++i)
#pragma unroll
        for (int j = 0; j < TN; ++j) { cr[i][j][0] = cr[i][j][1] = 0.0; ci[i][j][0] = ci[i][j][1] = 0.0; }
    int s = 0, s_prev = -1; uint32_t ph = 0;
    for (int c = 0; c < nchunks; ++c) {
        mbar_wait(full + s, ph);
        const double* a_base = As + ((size_t)s * KC + t) * LDA + g;
        const double2* b_base = Bs + ((size_t)s * KC + (t & 2)) * LDB + warp * TN * 8 + g;     // row of a; b is the next row
#pragma unroll
        for (int k4 = 0; k4 < KS; ++k4) {
            double av[TM];
            double2 ba[TN], bb[TN];
#pragma unroll
            for (int i = 0; i < TM; ++i) av[i] = a_base[(size_t)k4 * 4 * LDA + i * 8];
#pragma unroll
            for (int j = 0; j < TN; ++j) {
                ba[j] = b_base[(size_t)k4 * 4 * LDB + j * 8];
                bb[j] = b_base[(size_t)(k4 * 4 + 1) * LDB + j * 8];
            }
#pragma unroll
            for (int j = 0; j < TN; ++j) {
                const double x = fma(sig, bb[j].x, ba[j].x), y = fma(sig, bb[j].y, ba[j].y);     // a +- b
                const double bre = (t & 1) ? neg(y) : x, bim = (t & 1) ? x : y;                  // odd rows: times i
#pragma unroll
                for (int i = 0; i < TM; ++i) {
                    dmma884(cr[i][j][0], cr[i][j][1], av[i], bre);
                    dmma884(ci[i][j][0], ci[i][j][1], av[i], bim);
                }
            }
        }
        // release the PREVIOUS stage (see k_contract: an LDS still in flight must not race the next bulk copy)
        __syncwarp();
        if (lane == 0 && s_prev >= 0) mbar_arrive(empty + s_prev);
        s_prev = s;
        if (++s == ST) { s = 0; ph ^= 1u; }
    }
#pragma unroll
    for (int i = 0; i < TM; ++i) {
        const int m = i * 8 + g;
        if (m >= M) continue;
#pragma unroll
        for (int j = 0; j < TN; ++j) {
            const int n = n0 + warp * TN * 8 + j * 8 + 2 * t;
            double2* dst = T + (size_t)m * ldc + (size_t)p * X + n;
            if (n < X) dst[0] = make_double2(cr[i][j][0], ci[i][j][0]);
            if (n + 1 < X) dst[1] = make_double2(cr[i][j][1], ci[i][j][1]);
        }
    }
}

}  // namespace pe
