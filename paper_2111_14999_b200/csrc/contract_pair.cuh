// contract_pair.cuh -- step a4 (Eq. 70) with the +R / -R pairs of the phonon lattice vectors folded:
//     C[q][n] = sum_p w_p e^{i th_p(q)} g1'[p][n],      th_p = 2 pi q.Rp_p,  w_p = 1/deg_p[p]
// Lattice-vector lists come in inversion pairs (Wigner-Seitz supercells, full grids: Eq. 87):
// for Rp_pbar = -Rp_p with the same weight,
//     w e^{i th} a + w e^{-i th} b = (w cos th) (a + b) + (w sin th) (i (a - b)),        a = g1'[p], b = g1'[pbar]
// so the complex x complex GEMM over nRp rows becomes a REAL x complex GEMM over Kr rows,
//     A[q][r] = w cos th | w sin th      B[r][n] = a + b | i (a - b)       (R = 0: one row, A = w, B = a;
//                                                                            a vector without partner: b = 0, two rows)
// Kr = nRp for a symmetric list.  Real x complex = two real products sharing A: 4 real flop per (q, row, n) instead of
// 6 (three-multiply) or 8 (four-multiply) -- exact complex arithmetic, no normwise-only accuracy, and a third of the
// phase bytes (one real plane instead of three).  The host uses this form when 4 Kr < 6 nRp.
//
// Same pipeline as k_contract_planar (persistent CTAs, producer warp + TMA bulk-copy ring + mbarriers, FP64 DMMA
// consumers with row-interleaved tiles fed by LDS.128, stage release one chunk late, panel-major tile order).
//   AtR [KrPad][ldq]              real, row r, q contiguous (rows >= Kr and columns >= nq zero)
//   BP2 [Kr][ceil(N/64)][2][64]   planes re, im of B, blocked by 64 columns
// Shared row strides 68 / 132 doubles = 32 B mod 128 B: the 8 lanes of an LDS.128 quarter-warp fall into 8 distinct
// 16-byte slots.  Per k-step and warp (32 x 16 complex tile): 4 LDS.128, 16 DMMA (planar three-multiply: 9, 24).
#pragma once
#include "ptx_helpers.cuh"

// Rows per ring stage: 32 (ring = 4 x 32 x 1600 B = 200 KB, one CTA per SM).  Measured on the 4-atom cell: KC = 16 runs
// the stacked launch in 34.55 ms (91.3 % of the FP64 peak), KC = 32 in 33.26 ms (94.8 %): with 16 instead of 24 DMMA per
// k-step the per-chunk barrier traffic weighs more than in the planar kernel; two CTAs per SM at KC = 16: no change.
#ifndef PHOEBE_PAIR_KC
#define PHOEBE_PAIR_KC 32
#endif
#ifndef PHOEBE_PAIR_STAGES
#define PHOEBE_PAIR_STAGES 4
#endif

namespace pe {

struct PairCfg {
    static constexpr int BM = 64, BN = 64, WARPS_M = 2, WARPS_N = 4, KC = PHOEBE_PAIR_KC, STAGES = PHOEBE_PAIR_STAGES;
    static constexpr int kConsumerWarps = WARPS_M * WARPS_N;
    static constexpr int kThreads = (kConsumerWarps + 1) * 32;
    static constexpr int TM = 4, TN = 2;
    static constexpr int ROWA = 64, ROWB = 128;     // doubles of one operand row of a tile
    static constexpr int LDA = ROWA + 4, LDB = ROWB + 4;
    static constexpr size_t kRingBytes = (size_t)STAGES * KC * (LDA + LDB) * sizeof(double);
    static constexpr size_t kSmemBytes = kRingBytes + 2 * STAGES * sizeof(uint64_t);
    // q <-> -q fold (qfold.cuh): three ring stages + a lane-private copy of the accumulators (the even part Ce of a tile
    // while the odd part Co is summed): 8 warps x 32 lanes x 32 doubles
    static constexpr int FOLD_STAGES = 3;
    static constexpr size_t kFoldRingBytes = (size_t)FOLD_STAGES * KC * (LDA + LDB) * sizeof(double);
    static constexpr size_t kFoldSaveBytes = (size_t)kConsumerWarps * 32 * TM * TN * 2 * 2 * sizeof(double);
    static constexpr size_t kFoldSmemBytes = kFoldRingBytes + kFoldSaveBytes + 2 * FOLD_STAGES * sizeof(uint64_t);
};

// B rows from the canonical g1' [nRp][ld] (+ slot stride): row r = a + b (kind 0) or i (a - b) (kind 1),
// a = g1'[pa[r]], b = g1'[pb[r]] (pb < 0: b = 0).  grid (ntile, Kr, nslots), block 64; columns >= ncols are written 0.
__global__ void __launch_bounds__(64)
k_pack_pair(const double2* __restrict__ src, long long ld, long long strideS, int ncols, const int* __restrict__ pa,
            const int* __restrict__ pb, const int* __restrict__ kind, double* __restrict__ dst, long long strideD)
{
    const int c = threadIdx.x, tile = blockIdx.x, r = blockIdx.y, slot = blockIdx.z;
    const int n = tile * 64 + c;
    double2 v = make_double2(0.0, 0.0);
    if (n < ncols) {
        const double2* s = src + (size_t)slot * strideS + n;
        const double2 a = s[(size_t)pa[r] * ld];
        const int ib = pb[r];
        const double2 b = ib >= 0 ? s[(size_t)ib * ld] : make_double2(0.0, 0.0);
        if (kind[r] == 0) v = make_double2(a.x + b.x, a.y + b.y);
        else if (kind[r] == 1) v = make_double2(-(a.y - b.y), a.x - b.x);
        else v = make_double2(0.0, 0.0);                       // padding row between the cosine and the sine block
    }
    double* d = dst + (size_t)slot * strideD + ((size_t)r * gridDim.x + tile) * PairCfg::ROWB + c;
    d[0] = v.x; d[64] = v.y;
}

// Row order of the pair form (host contract, phoebe_elph_setup): a COSINE block -- one row per (+R, -R) pair or
// partner-less vector (K2 of them), then one per self-inverse vector (R = 0), zero rows up to a multiple of 4 (Kc4) --
// followed by the SINE block, one row per pair in the same order: row Kc4 + sl belongs to cosine row sl.  The cosine
// rows are even in q and the sine rows odd, which is what the q <-> -q fold below uses.
//
// A rows: AtR[r][col] = w[r] * cos(2 pi q . R[r]) (r < Kc) or w * sgn * sin(2 pi q . R[r - Kc4]); zero for padding rows and
// for columns >= nq.  One sincospi serves both rows of a pair.  blockIdx.y strides over cosine rows.
// qidx != nullptr: column col takes q-point qidx[col] (the representatives of the q <-> -q fold), and the number of
// columns is *ncol_dev; `run` (device flag, may be nullptr) == 0 makes the launch a no-op.
__global__ void __launch_bounds__(256)
k_qphase_pair(const double* __restrict__ q /* [nq][3] */, const double* __restrict__ Rrow /* [Kc][3] */,
              const double* __restrict__ wrow, int K2, int Kc, int Kc4, int nq, int Kr, int KrPad, int ldq,
              double sgn, double* __restrict__ AtR /* [KrPad][ldq] */, const int* __restrict__ qidx,
              const int* __restrict__ ncol_dev, const int* __restrict__ run, int run_when)
{
    if (run != nullptr && (*run != 0) != (run_when != 0)) return;
    const int col = blockIdx.x * blockDim.x + threadIdx.x;
    if (col >= ldq) return;
    if (ncol_dev != nullptr) nq = *ncol_dev;
    double q0 = 0.0, q1 = 0.0, q2 = 0.0;
    const bool valid = col < nq;
    if (valid) {
        const size_t iq = qidx != nullptr ? (size_t)qidx[col] : (size_t)col;
        q0 = q[3 * iq]; q1 = q[3 * iq + 1]; q2 = q[3 * iq + 2];
    }
    for (int r = blockIdx.y; r < Kc4; r += gridDim.y) {
        double vc = 0.0, vs = 0.0;
        if (valid && r < Kc) {
            const double x = q0 * Rrow[3 * r] + q1 * Rrow[3 * r + 1] + q2 * Rrow[3 * r + 2];
            double sn, cs;
            sincospi(2.0 * x, &sn, &cs);
            vc = wrow[r] * cs; vs = wrow[r] * sgn * sn;
        }
        AtR[(size_t)r * ldq + col] = vc;
        if (r < K2) AtR[(size_t)(Kc4 + r) * ldq + col] = vs;
    }
    for (int r = Kr + blockIdx.y; r < KrPad; r += gridDim.y) AtR[(size_t)r * ldq + col] = 0.0;
}

// AtR, BP2 as above (BP2 of k slot 0; slot j at + j*strideBslot doubles); C [M][ldc] complex; K = Kr, Kpad = KrPad.
// rowsPerB > 0: rows [j*rowsPerB, (j+1)*rowsPerB) of the stacked q lists use slot j (multi-k form, see k_contract).
//
// fold.meta != nullptr (qfold.cuh): meta[0] = representatives, meta[1] = whether the q <-> -q fold is taken.
//   FOLD = false: the plain launch returns at once when the fold is taken.
//   FOLD = true : returns at once when it is not; else M = meta[0] rows (the columns of AtR are the representatives), the
//   accumulators are saved at the cosine | sine boundary (row Kc4) and the tile is finished as
//   C[rep] = Ce + Co, C[mate] = Ce - Co.
struct FoldArgs { const int* meta; const int* rep_idx; const int* mate; int Kc4; };

template <bool FOLD>
__global__ void __launch_bounds__(PairCfg::kThreads, 1)
k_contract_pair(const double* __restrict__ AtR, int lda, const double* __restrict__ BP2, int ntnB, long long strideBslot,
                double2* __restrict__ C, long long ldc, int M, int N, int K, int Kpad, int rowsPerB, int rowOffset,
                int panelW, CMap cm, FoldArgs fold)
{
    using Cfg = PairCfg;
    constexpr int BM = Cfg::BM, BN = Cfg::BN, KC = Cfg::KC, STAGES = FOLD ? Cfg::FOLD_STAGES : Cfg::STAGES;
    constexpr int LDA = Cfg::LDA, LDB = Cfg::LDB;
    constexpr int ROWA = Cfg::ROWA, ROWB = Cfg::ROWB, TM = Cfg::TM, TN = Cfg::TN, KS = KC / 4;
    constexpr size_t kRingBytes = FOLD ? Cfg::kFoldRingBytes : Cfg::kRingBytes;
    if (fold.meta != nullptr) {
        if ((fold.meta[1] != 0) != FOLD) return;
        if (FOLD) M = fold.meta[0];
    }
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* As = reinterpret_cast<double*>(smem_raw);                    // [STAGES][KC][LDA]
    double* Bs = As + (size_t)STAGES * KC * LDA;                         // [STAGES][KC][LDB]
    double* save = Bs + (size_t)STAGES * KC * LDB;                       // FOLD: [32 accumulator values][256 consumer lanes]
    uint64_t* full = reinterpret_cast<uint64_t*>(save + (FOLD ? Cfg::kFoldSaveBytes / sizeof(double) : 0));
    uint64_t* empty = full + STAGES;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int i = threadIdx.x; i < (int)(kRingBytes / sizeof(double2)); i += Cfg::kThreads)
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
        // ---------------- producer warp: a 512-byte (A) and a 1024-byte (B) bulk copy per operand row ----------------
        int s = 0; uint32_t ph = 0;
        for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            int tm, tn;
            decode(tile, tm, tn);
            const double* a_src = AtR + (size_t)tm * ROWA;
            const double* b_src = BP2 + (size_t)tn * ROWB +
                                  (rowsPerB > 0 ? (size_t)((rowOffset + tm * BM) / rowsPerB) * strideBslot : (size_t)0);
            for (int c = 0; c < nchunks; ++c) {
                mbar_wait(empty + s, ph ^ 1u);
                const int k0 = c * KC;
                const int rows_b = max(0, min(KC, K - k0));
                if (lane == 0)
                    mbar_arrive_expect_tx(full + s, (uint32_t)((KC * ROWA + rows_b * ROWB) * sizeof(double)));
                __syncwarp();
                if (lane < KC)
                    bulk_g2s(As + ((size_t)s * KC + lane) * LDA, a_src + (size_t)(k0 + lane) * lda,
                             ROWA * sizeof(double), full + s);
                if (lane < rows_b)
                    bulk_g2s(Bs + ((size_t)s * KC + lane) * LDB, b_src + (size_t)(k0 + lane) * ntnB * ROWB,
                             ROWB * sizeof(double), full + s);
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
        double cr[TM][TN][2], ci[TM][TN][2];               // Re C = sum A * Re B,  Im C = sum A * Im B
#pragma unroll
        for (int i = 0; i < TM; ++i)
#pragma unroll
            for (int j = 0; j < TN; ++j)
#pragma unroll
                for (int h = 0; h < 2; ++h) { cr[i][j][h] = 0.0; ci[i][j][h] = 0.0; }

        for (int c = 0; c < nchunks; ++c) {
            mbar_wait(full + s, ph);
            const double* a_base = As + ((size_t)s * KC + t) * LDA + wm * 32 + 2 * g;
            const double* b_base = Bs + ((size_t)s * KC + t) * LDB + wn * 16 + 2 * g;
            auto lda2 = [&](int k4, int ip) {
                return *reinterpret_cast<const double2*>(a_base + (size_t)k4 * 4 * LDA + ip * 16);
            };
            auto ldb2 = [&](int k4, int plane) {
                return *reinterpret_cast<const double2*>(b_base + (size_t)k4 * 4 * LDB + plane * 64);
            };
            double2 a[2][2], b[2][2];               // [register buffer][pair | plane]: .x = even tile, .y = odd tile
            a[0][0] = lda2(0, 0); a[0][1] = lda2(0, 1); b[0][0] = ldb2(0, 0); b[0][1] = ldb2(0, 1);
            // the last chunk runs only the k-steps that hold rows < K, a warp-uniform branch
            const int ks_n = min(KS, (K + 3 - c * KC) >> 2);
#pragma unroll
            for (int k4 = 0; k4 < KS; ++k4) {
                const int cur = k4 & 1, nxt = cur ^ 1;
                if (k4 >= ks_n) break;
                if (FOLD && c * KC + 4 * k4 == fold.Kc4) {
                    // cosine | sine boundary: keep the even part Ce of the tile (lane-private slots), start the odd part
#pragma unroll
                    for (int i = 0; i < TM; ++i)
#pragma unroll
                        for (int j = 0; j < TN; ++j)
#pragma unroll
                            for (int h = 0; h < 2; ++h) {
                                const int e = ((i * TN + j) * 2 + h) * 2;
                                save[(size_t)e * 256 + threadIdx.x] = cr[i][j][h];
                                save[(size_t)(e + 1) * 256 + threadIdx.x] = ci[i][j][h];
                                cr[i][j][h] = 0.0; ci[i][j][h] = 0.0;
                            }
                }
                if (k4 + 1 < KS) {
                    a[nxt][0] = lda2(k4 + 1, 0); a[nxt][1] = lda2(k4 + 1, 1);
                    b[nxt][0] = ldb2(k4 + 1, 0); b[nxt][1] = ldb2(k4 + 1, 1);
                }
#pragma unroll
                for (int i = 0; i < TM; ++i) {
                    const double av = (i & 1) ? a[cur][i >> 1].y : a[cur][i >> 1].x;
#pragma unroll
                    for (int j = 0; j < TN; ++j) {
                        const double br = j ? b[cur][0].y : b[cur][0].x;
                        const double bi = j ? b[cur][1].y : b[cur][1].x;
                        dmma884(cr[i][j][0], cr[i][j][1], av, br);
                        dmma884(ci[i][j][0], ci[i][j][1], av, bi);
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
            if (FOLD) {
                double2* dst = C + (size_t)fold.rep_idx[m] * ldc;
                const int im = fold.mate[m];
                double2* dstm = C + (size_t)max(im, 0) * ldc;
#pragma unroll
                for (int cc = 0; cc < 4; ++cc) {
                    const int j = cc & 1, h = cc >> 1;
                    const int e = ((i * TN + j) * 2 + h) * 2;
                    const double er = save[(size_t)e * 256 + threadIdx.x], ei = save[(size_t)(e + 1) * 256 + threadIdx.x];
                    if (cc < nleft) {
                        dst[coff[cc]] = make_double2(er + cr[i][j][h], ei + ci[i][j][h]);
                        if (im >= 0) dstm[coff[cc]] = make_double2(er - cr[i][j][h], ei - ci[i][j][h]);
                    }
                }
                continue;
            }
            double2* dst = C + (size_t)m * ldc;
#pragma unroll
            for (int cc = 0; cc < 4; ++cc) {
                const int j = cc & 1, h = cc >> 1;
                if (cc < nleft) dst[coff[cc]] = make_double2(cr[i][j][h], ci[i][j][h]);
            }
        }
    }
}

}  // namespace pe
