// contract_planar.cuh -- step a4 (Eq. 70), the planar-operand form of the Rp contraction:
//     C[q][n] = sum_p Pt[p][q] * g1'[p][n]                 (complex128, three-multiply product)
//
// Same pipeline as k_contract (persistent CTAs, producer warp + TMA bulk-copy ring + mbarriers, FP64 DMMA consumers,
// stage release one chunk late, panel-major tile order) but the operands arrive PLANAR and BLOCKED:
//     PtP [Kpad][ldq/64][3][64]   g1P [nRp][ceil(N/64)][3][64]      planes: 0 = re, 1 = im, 2 = re + im
// so that (i) the operand sums of the three-multiply product are data, not DADDs, and (ii) ONE LDS.128 of a plane
// feeds TWO DMMA tiles: the two doubles a lane loads are column c and c+1 of the tile row block, and the tiles are
// DEFINED to interleave -- tile 2i takes the even, tile 2i+1 the odd rows (columns for B) of a 16-wide block.  Any
// assignment of rows to tiles is a valid GEMM tiling; only the C store has to follow it.
// Why: every LDS / DADD that ptxas lets overwrite a fragment register right behind a DMMA costs about as much as a
// DMMA on B200; this form issues 9 such instructions per k-step instead of 12
// (6 LDS.128 + 6 DADD), measured 3.20 ms vs 3.44 ms per 8192-q launch of the 4-atom cell.
//
// Fragment geometry (BM = BN = 64, 8 consumer warps as 2 (m) x 4 (n), warp tile 32 x 16 = TM 4 x TN 2 DMMA tiles):
//   A: lane (g,t) loads plane[k0+t][mw + 16*ip + 2g .. +1]   -> tile i = 2*ip   row g  <-> m = mw + 16*ip + 2g
//                                                              tile i = 2*ip+1 row g  <-> m = mw + 16*ip + 2g + 1
//   B: lane (g,t) loads plane[k0+t][nw + 2g .. +1]           -> tile j = 0 col g <-> n = nw + 2g, j = 1 <-> n = nw + 2g + 1
//   C accumulator of tile (i,j), lane (g,t): rows g, cols 2t, 2t+1 of the tile
//       -> m = mw + 16*(i/2) + 2g + (i&1),   n = nw + 4t + (j&1)  and  nw + 4t + 2 + (j&1)
//      i.e. a lane owns 4 CONSECUTIVE complex columns n = nw + 4t .. 4t+3 of each of its rows (64-byte stores).
// Shared row stride = 3*64 + 4 doubles = 1568 B = 32 B mod 128 B: the 8 lanes of an LDS.128 quarter-warp
// (g = 0,1 x t = 0..3) fall into 8 distinct 16-byte slots -- conflict-free.
#pragma once
#include "ptx_helpers.cuh"

namespace pe {

struct PlanarCfg {
    static constexpr int BM = 64, BN = 64, WARPS_M = 2, WARPS_N = 4, KC = 16, STAGES = 4;
    static constexpr int kConsumerWarps = WARPS_M * WARPS_N;
    static constexpr int kThreads = (kConsumerWarps + 1) * 32;
    static constexpr int TM = 4, TN = 2;
    static constexpr int ROW = 3 * 64;              // doubles of one blocked row: [3 planes][64]
    static constexpr int LDP = ROW + 4;             // shared row stride in doubles
    static constexpr size_t kRingBytes = (size_t)STAGES * KC * 2 * LDP * sizeof(double);
    static constexpr size_t kSmemBytes = kRingBytes + 2 * STAGES * sizeof(uint64_t);
};

// canonical complex [rows][ld] (+ slot stride) -> planar blocked [rows][ntile][3][64]; columns >= ncols are written 0.
// grid (ntile, rows, nslots), block 64.
__global__ void __launch_bounds__(64)
k_pack_planar(const double2* __restrict__ src, long long ld, long long strideS, int ncols,
              double* __restrict__ dst, long long strideD)
{
    const int c = threadIdx.x, tile = blockIdx.x, row = blockIdx.y, slot = blockIdx.z;
    const int n = tile * 64 + c;
    double2 v = make_double2(0.0, 0.0);
    if (n < ncols) v = src[(size_t)slot * strideS + (size_t)row * ld + n];
    double* d = dst + (size_t)slot * strideD + ((size_t)row * gridDim.x + tile) * PlanarCfg::ROW + c;
    d[0] = v.x; d[64] = v.y; d[128] = v.x + v.y;
}

// AtP: planar blocked phases [Kpad][ntmA][3][64] (rows K..Kpad-1 and columns >= M zero);  BP: planar blocked g1'
// [K][ntnB][3][64] of k slot 0, slot j at + j*strideBslot doubles;  C [M][ldc] complex.
// rowsPerB > 0: rows [j*rowsPerB, (j+1)*rowsPerB) of the stacked q lists use slot j (multi-k form, see k_contract).
__global__ void __launch_bounds__(PlanarCfg::kThreads, 1)
k_contract_planar(const double* __restrict__ AtP, int ntmA, const double* __restrict__ BP, int ntnB,
                  long long strideBslot, double2* __restrict__ C, long long ldc, int M, int N, int K, int Kpad,
                  int rowsPerB, int rowOffset, int panelW, CMap cm)
{
    using Cfg = PlanarCfg;
    constexpr int BM = Cfg::BM, BN = Cfg::BN, KC = Cfg::KC, STAGES = Cfg::STAGES, LDP = Cfg::LDP, ROW = Cfg::ROW;
    constexpr int TM = Cfg::TM, TN = Cfg::TN, KS = KC / 4;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* As = reinterpret_cast<double*>(smem_raw);                    // [STAGES][KC][LDP]
    double* Bs = As + (size_t)STAGES * KC * LDP;                         // [STAGES][KC][LDP]
    uint64_t* full = reinterpret_cast<uint64_t*>(Bs + (size_t)STAGES * KC * LDP);
    uint64_t* empty = full + STAGES;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int i = threadIdx.x; i < (int)(Cfg::kRingBytes / sizeof(double2)); i += Cfg::kThreads)
        reinterpret_cast<double2*>(As)[i] = make_double2(0.0, 0.0);
    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, Cfg::kConsumerWarps); }
        mbar_fence_init();
    }
    fence_proxy_async();
    __syncthreads();
    const int nchunks = Kpad / KC;
    const int ntn = (N + BN - 1) / BN, ntm = (M + BM - 1) / BM;
    const int ntiles = ntn * ntm;
    auto decode = [&](int tile, int& tm, int& tn) {        // panel-major order, see k_contract
        const int pw = min(panelW, ntn);
        const int panel = tile / (pw * ntm);
        const int w = min(pw, ntn - panel * pw);
        const int rr = tile - panel * pw * ntm;
        tm = rr / w;
        tn = panel * pw + rr - tm * w;
    };

    if (warp == Cfg::kConsumerWarps) {
        // ---------------- producer warp: one 1536-byte bulk copy per operand row ----------------
        int s = 0; uint32_t ph = 0;
        for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            int tm, tn;
            decode(tile, tm, tn);
            const double* a_src = AtP + (size_t)tm * ROW;
            const double* b_src = BP + (size_t)tn * ROW +
                                  (rowsPerB > 0 ? (size_t)((rowOffset + tm * BM) / rowsPerB) * strideBslot : (size_t)0);
            for (int c = 0; c < nchunks; ++c) {
                mbar_wait(empty + s, ph ^ 1u);
                const int k0 = c * KC;
                const int rows_b = max(0, min(KC, K - k0));
                if (lane == 0) mbar_arrive_expect_tx(full + s, (uint32_t)((KC + rows_b) * ROW * sizeof(double)));
                __syncwarp();
                if (lane < KC)
                    bulk_g2s(As + ((size_t)s * KC + lane) * LDP, a_src + (size_t)(k0 + lane) * ntmA * ROW,
                             ROW * sizeof(double), full + s);
                if (lane < rows_b)
                    bulk_g2s(Bs + ((size_t)s * KC + lane) * LDP, b_src + (size_t)(k0 + lane) * ntnB * ROW,
                             ROW * sizeof(double), full + s);
                if (++s == STAGES) { s = 0; ph ^= 1u; }
            }
        }
        return;
    }

    // ---------------- consumer warps ----------------
    const int wm = warp / Cfg::WARPS_N, wn = warp % Cfg::WARPS_N;
    const int g = lane >> 2, t = lane & 3;
    int s = 0, s_prev = -1; uint32_t ph = 0;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        int tm, tn;
        decode(tile, tm, tn);
        const int n0 = tn * BN, m0 = tm * BM;
        // T1 = sum Ar*Br, T2 = sum Ai*Bi, T3 = sum (Ar+Ai)*(Br+Bi);  Re C = T1 - T2, Im C = T3 - T1 - T2
        double cr[TM][TN][2], ci[TM][TN][2], cs[TM][TN][2];
#pragma unroll
        for (int i = 0; i < TM; ++i)
#pragma unroll
            for (int j = 0; j < TN; ++j)
#pragma unroll
                for (int h = 0; h < 2; ++h) { cr[i][j][h] = 0.0; ci[i][j][h] = 0.0; cs[i][j][h] = 0.0; }

        for (int c = 0; c < nchunks; ++c) {
            mbar_wait(full + s, ph);
            const double* a_base = As + ((size_t)s * KC + t) * LDP + wm * 32 + 2 * g;
            const double* b_base = Bs + ((size_t)s * KC + t) * LDP + wn * 16 + 2 * g;
            auto lda2 = [&](int k4, int plane, int ip) {
                return *reinterpret_cast<const double2*>(a_base + (size_t)k4 * 4 * LDP + plane * 64 + ip * 16);
            };
            auto ldb2 = [&](int k4, int plane) {
                return *reinterpret_cast<const double2*>(b_base + (size_t)k4 * 4 * LDP + plane * 64);
            };
            double2 a[2][3][2], b[2][3];            // [register buffer][plane][pair]: .x = even tile, .y = odd tile
#pragma unroll
            for (int pl = 0; pl < 3; ++pl) {
                a[0][pl][0] = lda2(0, pl, 0); a[0][pl][1] = lda2(0, pl, 1); b[0][pl] = ldb2(0, pl);
            }
            // the last chunk runs only the k-steps that hold rows < K (K = 343: 2 of 4), a warp-uniform branch
            const int ks_n = min(KS, (K + 3 - c * KC) >> 2);
#pragma unroll
            for (int k4 = 0; k4 < KS; ++k4) {
                const int cur = k4 & 1, nxt = cur ^ 1;
                if (k4 >= ks_n) break;
                if (k4 + 1 < KS) {
#pragma unroll
                    for (int pl = 0; pl < 3; ++pl) {
                        a[nxt][pl][0] = lda2(k4 + 1, pl, 0); a[nxt][pl][1] = lda2(k4 + 1, pl, 1); b[nxt][pl] = ldb2(k4 + 1, pl);
                    }
                }
#pragma unroll
                for (int i = 0; i < TM; ++i) {
                    const int ip = i >> 1;
                    const double ar = (i & 1) ? a[cur][0][ip].y : a[cur][0][ip].x;
                    const double ai = (i & 1) ? a[cur][1][ip].y : a[cur][1][ip].x;
                    const double as = (i & 1) ? a[cur][2][ip].y : a[cur][2][ip].x;
#pragma unroll
                    for (int j = 0; j < TN; ++j) {
                        const double br = j ? b[cur][0].y : b[cur][0].x;
                        const double bi = j ? b[cur][1].y : b[cur][1].x;
                        const double bs = j ? b[cur][2].y : b[cur][2].x;
                        dmma884(cr[i][j][0], cr[i][j][1], ar, br);
                        dmma884(ci[i][j][0], ci[i][j][1], ai, bi);
                        dmma884(cs[i][j][0], cs[i][j][1], as, bs);
                    }
                }
            }
            // release the PREVIOUS stage (see k_contract: an LDS still in flight must not race the next bulk copy)
            __syncwarp();
            if (lane == 0 && s_prev >= 0) mbar_arrive(empty + s_prev);
            s_prev = s;
            if (++s == STAGES) { s = 0; ph ^= 1u; }
        }

        // ---------------- store C: a lane owns 4 consecutive columns of each of its 4 rows ----------------
        const int nleft = N - (n0 + wn * 16 + 4 * t);
        long long coff[4];                                  // where the rotation kernel wants them (CMap)
#pragma unroll
        for (int cc = 0; cc < 4; ++cc) coff[cc] = cc < nleft ? cmap_off(n0 + wn * 16 + 4 * t + cc, cm) : 0;
#pragma unroll
        for (int i = 0; i < TM; ++i) {
            const int m = m0 + wm * 32 + 16 * (i >> 1) + 2 * g + (i & 1);
            if (m >= M) continue;
            double2* dst = C + (size_t)m * ldc;
#pragma unroll
            for (int cc = 0; cc < 4; ++cc) {
                const int j = cc & 1, h = cc >> 1;
                const double t1 = cr[i][j][h], t2 = ci[i][j][h];
                if (cc < nleft) dst[coff[cc]] = make_double2(t1 - t2, cs[i][j][h] - t1 - t2);
            }
        }
    }
}

}  // namespace pe
