// qbatch_kernels.cuh -- steps a3..a7 (Eq. 70 + Eq. 7): completion for a batch of q.
//
//   a3  Pt[p][q]           = e^{2 pi i q.Rp_p}/deg_p[p]                      (k_qphase)
//   a4  C[q][n]            = sum_p Pt[p][q] g1[p][n]      n=(b1,w2,kappa)     (k_contract, FP64 DMMA)
//   a5  D[q][b1][b2][ka]   = sum_w2 conj(Ukq[q][w2][b2]) C[q][b1][w2][ka]     (k_rotate_epilogue)
//   a6  E[q][b1][b2][nu]   = sum_ka D[q][b1][b2][ka] ev[q][ka][nu]
//   a7  out                = |E|^2/(2 omega)   (0 where omega <= 0)
#pragma once
#include "ptx_helpers.cuh"
#include "rot_args.cuh"

namespace pe {

// ---------------------------------------------------------------------------
// a3: phases, written TRANSPOSED (p-major, q contiguous) so that both operands of
// the contraction are "k-major" and a tile row is one contiguous bulk copy.
// Columns q in [nq, ldq) and rows p in [nRp, Kpad) are written as zeros.
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_qphase(const double* __restrict__ q /* [nq][3] */, const double* __restrict__ Rp, const double* __restrict__ deg_p,
         int nq, int nRp, int Kpad, int ldq, double2* __restrict__ Pt /* [Kpad][ldq] */,
         double sgn /* +1: e^{+2 pi i q.R} (Eq. 13); -1: e^{-2 pi i q.R} (Eq. 5, set_conventions) */,
         double* __restrict__ PtP /* planar blocked copy [Kpad][ldq/64][3][64] for k_contract_planar, or nullptr */)
{
    const int iq = blockIdx.x * blockDim.x + threadIdx.x;
    if (iq >= ldq) return;
    double q0 = 0.0, q1 = 0.0, q2 = 0.0;
    const bool valid = iq < nq;
    if (valid) { q0 = q[3 * (size_t)iq]; q1 = q[3 * (size_t)iq + 1]; q2 = q[3 * (size_t)iq + 2]; }
    for (int p = blockIdx.y; p < Kpad; p += gridDim.y) {
        double2 v = make_double2(0.0, 0.0);
        if (valid && p < nRp) {
            const double x = q0 * Rp[3 * p] + q1 * Rp[3 * p + 1] + q2 * Rp[3 * p + 2];
            double sn, cs;
            sincospi(2.0 * x, &sn, &cs);
            const double w = 1.0 / deg_p[p];
            v = make_double2(cs * w, sgn * sn * w);
        }
        if (PtP) {
            double* d = PtP + ((size_t)p * (ldq >> 6) + (iq >> 6)) * 192 + (iq & 63);
            d[0] = v.x; d[64] = v.y; d[128] = v.x + v.y;
        } else {
            Pt[(size_t)p * ldq + iq] = v;
        }
    }
}

// ---------------------------------------------------------------------------
// f4: the (q, nu)-only factor of the polar long-range term (Eq. 15):
//   P[q][nu] = i coeff sum_G (Q . Zeff_nu) / (Q . eps_inf . Q),  Q = (q + G) . recip,
//   Zeff_nu[a] = sum_{s,b} Z*_s[a][b] ev[q][3s+b][nu]
// The G sum does not depend on nu: V[a] = sum_G Q_a / (Q.eps.Q) (real), W[3s+b] = sum_a V_a Z*_s[a][b],
// P[nu] = i coeff sum_kappa W[kappa] ev[kappa][nu].  One warp per q; lanes stride over G, fixed-order
// shuffle reduction; the term with Q exactly zero (G = -q) is skipped.
// ---------------------------------------------------------------------------
struct PolarParams { double recip[9]; double eps[9]; double coeff; };

__global__ void __launch_bounds__(128)
k_polar_amp(const double* __restrict__ q /* [nq][3] */, const double2* __restrict__ ev /* [nq][nm][nm] */,
            const double* __restrict__ G /* [nG][3] */, const double* __restrict__ Zstar /* [nm/3][3][3] */,
            int nq, int nm, int nG, PolarParams pp, double2* __restrict__ P /* [nq][nm] */)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double* W = reinterpret_cast<double*>(smem_raw) + (size_t)warp * nm;      // [warps][nm]
    const int iq = blockIdx.x * (blockDim.x >> 5) + warp;
    if (iq >= nq) return;
    const double q0 = q[3 * (size_t)iq], q1 = q[3 * (size_t)iq + 1], q2 = q[3 * (size_t)iq + 2];
    double v0 = 0.0, v1 = 0.0, v2 = 0.0;
    for (int ig = lane; ig < nG; ig += 32) {
        const double c0 = q0 + G[3 * ig], c1 = q1 + G[3 * ig + 1], c2 = q2 + G[3 * ig + 2];
        const double Q0 = c0 * pp.recip[0] + c1 * pp.recip[3] + c2 * pp.recip[6];
        const double Q1 = c0 * pp.recip[1] + c1 * pp.recip[4] + c2 * pp.recip[7];
        const double Q2 = c0 * pp.recip[2] + c1 * pp.recip[5] + c2 * pp.recip[8];
        if (Q0 == 0.0 && Q1 == 0.0 && Q2 == 0.0) continue;
        const double den = Q0 * (pp.eps[0] * Q0 + pp.eps[1] * Q1 + pp.eps[2] * Q2) +
                           Q1 * (pp.eps[3] * Q0 + pp.eps[4] * Q1 + pp.eps[5] * Q2) +
                           Q2 * (pp.eps[6] * Q0 + pp.eps[7] * Q1 + pp.eps[8] * Q2);
        const double r = 1.0 / den;
        v0 = fma(Q0, r, v0); v1 = fma(Q1, r, v1); v2 = fma(Q2, r, v2);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        v0 += __shfl_xor_sync(0xffffffffu, v0, o);
        v1 += __shfl_xor_sync(0xffffffffu, v1, o);
        v2 += __shfl_xor_sync(0xffffffffu, v2, o);
    }
    for (int ka = lane; ka < nm; ka += 32) {
        const double* Z = Zstar + (size_t)(ka / 3) * 9 + (ka % 3);          // Z*_s[a][b], b = ka % 3
        W[ka] = v0 * Z[0] + v1 * Z[3] + v2 * Z[6];
    }
    __syncwarp();
    const double2* Zq = ev + (size_t)iq * nm * nm;
    for (int nu = lane; nu < nm; nu += 32) {
        double sr = 0.0, si = 0.0;
        for (int ka = 0; ka < nm; ++ka) {
            const double2 z = Zq[(size_t)ka * nm + nu];
            sr = fma(W[ka], z.x, sr); si = fma(W[ka], z.y, si);
        }
        P[(size_t)iq * nm + nu] = make_double2(-pp.coeff * si, pp.coeff * sr);     // i * coeff * (sr + i si)
    }
}

// ---------------------------------------------------------------------------
// a4 (and the multi-k form of a1): batched complex128 GEMM on the FP64 tensor cores
//     C_z[m][n] = sum_{k<K} At[k][m] * B_z[k][n]          z = blockIdx.z
// At is [Kpad][lda] (k-major, Kpad a multiple of KC, rows K..Kpad-1 and columns >= M zero), shared by all z;
// optionally B switches slab with the row block (rowsPerB, see the producer) -- the multi-k form of a4;
// B_z = B + z*strideB is [K][ldb] (k-major); C_z = C + z*strideC is [M][ldc].
//   a4:  At = Pt (phases of the q batch), B = g1' (K = nRp, N = nb1*nw*nm), C = C[q][n]
//   a1:  At = phases of a k batch, B_z = g_W[p=z] (K = nRe, N = nw*nw*nm), C_z = T[k][p][x]
//
// Warp-specialised: one producer warp streams [KC x BM] tiles of At and [KC x BN]
// tiles of B into a STAGES-deep shared-memory ring with TMA 1-D bulk copies
// (one per tile row, completion on an mbarrier); WARPS_M x WARPS_N consumer warps
// run FP64 tensor-core tiles (mma.sync m8n8k4 -> SASS DMMA.8x8x4):
//     Cr += Ar*Br + (-Ai)*Bi ,   Ci += Ar*Bi + Ai*Br          (4 DMMA per 8x8 complex tile per k4)
// Only valid data are copied (rows < K, columns < N); the ring is zeroed once so
// that what the padded k-steps / ragged columns read is finite and multiplies
// into discarded outputs or against the zero rows of At.
// Shared rows are padded by 2 complex so that the per-lane fragment loads
// (LDS.128 at [k0+t][.. + g]) are bank-conflict free.
// ---------------------------------------------------------------------------
template <int BM, int BN, int WARPS_M, int WARPS_N, int KC, int STAGES>
struct ContractCfg {
    static constexpr int kConsumerWarps = WARPS_M * WARPS_N;
    static constexpr int kThreads = (kConsumerWarps + 1) * 32;
    static constexpr int TM = BM / WARPS_M / 8;
    static constexpr int TN = BN / WARPS_N / 8;
    static constexpr int LDA = BM + 2;     // complex elements per shared row
    static constexpr int LDB = BN + 2;
    static constexpr size_t kRingBytes = (size_t)STAGES * KC * (LDA + LDB) * sizeof(double2);
    static constexpr size_t kSmemBytes = kRingBytes + 2 * STAGES * sizeof(uint64_t);
    static_assert(BM % (WARPS_M * 8) == 0 && BN % (WARPS_N * 8) == 0, "tile/warp mismatch");
    static_assert(KC % 4 == 0 && KC <= 32, "KC rows are issued by the 32 producer lanes");
};

template <int BM, int BN, int WARPS_M, int WARPS_N, int KC, int STAGES, bool M3, int MINB = 1>
__global__ void __launch_bounds__((WARPS_M * WARPS_N + 1) * 32, MINB)
k_contract(const double2* __restrict__ At, int lda, const double2* __restrict__ B, int ldb, long long strideB,
           double2* __restrict__ C, long long ldc, long long strideC, int M, int N, int K, int Kpad, int nbatch,
           int rowsPerB, int rowOffset, long long strideBrow, int panelW, CMap cm)
{
    using Cfg = ContractCfg<BM, BN, WARPS_M, WARPS_N, KC, STAGES>;
    constexpr int TM = Cfg::TM, TN = Cfg::TN, LDA = Cfg::LDA, LDB = Cfg::LDB;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double2* As = reinterpret_cast<double2*>(smem_raw);                  // [STAGES][KC][LDA]
    double2* Bs = As + (size_t)STAGES * KC * LDA;                        // [STAGES][KC][LDB]
    uint64_t* full = reinterpret_cast<uint64_t*>(Bs + (size_t)STAGES * KC * LDB);
    uint64_t* empty = full + STAGES;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int i = threadIdx.x; i < (int)(Cfg::kRingBytes / sizeof(double2)); i += Cfg::kThreads)
        As[i] = make_double2(0.0, 0.0);
    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, Cfg::kConsumerWarps); }
        mbar_fence_init();
    }
    fence_proxy_async();      // generic-proxy zero fill ordered before the async-proxy (TMA) writes
    __syncthreads();
    const int nchunks = Kpad / KC;          // host contract: Kpad % KC == 0, rows K..Kpad-1 of At are zero
    // PERSISTENT: the CTA walks tiles blockIdx.x, blockIdx.x + gridDim.x, ... (n fastest, then m, then batch z);
    // the ring and its barrier phases run on across tile boundaries, so the producer is already filling the
    // stages of the next tile while the consumers store C -- no per-tile prologue, no pipeline drain.
    const int ntn = (N + BN - 1) / BN, ntm = (M + BM - 1) / BM;
    const long long ntiles = (long long)ntn * ntm * nbatch;
    // Tile order inside a batch entry: panels of panelW column tiles, and inside a panel row block by row block
    // (tn fastest).  With panelW = gridDim.x every CTA of the persistent grid keeps ONE column tile for the whole
    // panel, so the panel of B (panelW x K x BN) stays in L2 while the row blocks of A stream through once per panel:
    // B is read from HBM once and A ceil(ntn/panelW) times, instead of B once per row block (ncu r1f, large cell:
    // 42.7 GB read per launch for 0.26 GB of operands).  panelW >= ntn gives the plain n-fastest order.
    auto decode = [&](long long tile, int& tm, int& tn, long long& z) {
        const long long per_z = (long long)ntn * ntm;
        z = tile / per_z;
        const int r = (int)(tile - z * per_z);
        const int pw = min(panelW, ntn);
        const int panel = r / (pw * ntm);
        const int w = min(pw, ntn - panel * pw);             // width of this (possibly last, narrower) panel
        const int rr = r - panel * pw * ntm;
        tm = rr / w;
        tn = panel * pw + rr - tm * w;
    };

    if (warp == Cfg::kConsumerWarps) {
        // ---------------- producer warp ----------------
        int s = 0; uint32_t ph = 0;
        for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            int tn, tm; long long z;
            decode(tile, tm, tn, z);
            const int n0 = tn * BN, m0 = tm * BM;
            const double2* a_src = At + m0;
            // rowsPerB > 0 (q batches of several k-points stacked along M): rows [j*rowsPerB, (j+1)*rowsPerB) of the
            // whole stack take the B of k slot j (host contract: rowsPerB and rowOffset are multiples of BM)
            const double2* b_src = B + (size_t)z * strideB + n0 +
                                   (rowsPerB > 0 ? (size_t)((rowOffset + m0) / rowsPerB) * strideBrow : (size_t)0);
            const int bn = min(BN, N - n0);                     // valid columns of this tile
            for (int c = 0; c < nchunks; ++c) {
                mbar_wait(empty + s, ph ^ 1u);
                const int k0 = c * KC;
                const int rows_b = max(0, min(KC, K - k0));
                if (lane == 0)
                    mbar_arrive_expect_tx(full + s, (uint32_t)((KC * BM + rows_b * bn) * sizeof(double2)));
                __syncwarp();
                if (lane < KC)
                    bulk_g2s(As + ((size_t)s * KC + lane) * LDA, a_src + (size_t)(k0 + lane) * lda,
                             BM * sizeof(double2), full + s);
                if (lane < rows_b)
                    bulk_g2s(Bs + ((size_t)s * KC + lane) * LDB, b_src + (size_t)(k0 + lane) * ldb,
                             bn * sizeof(double2), full + s);
                if (++s == STAGES) { s = 0; ph ^= 1u; }
            }
        }
        return;
    }

    // ---------------- consumer warps ----------------
    const int wm = warp / WARPS_N, wn = warp % WARPS_N;
    const int g = lane >> 2, t = lane & 3;
    // M3 = false: cr = Re C, ci = Im C (4 DMMA per tile and k-step).
    // M3 = true : the three-multiply complex product (3 DMMA per tile and k-step):
    //     cr = T1 = sum Ar*Br,  ci = T2 = sum Ai*Bi,  cs = T3 = sum (Ar+Ai)*(Br+Bi)
    //     Re C = T1 - T2,  Im C = T3 - T1 - T2     (formed once, after the k loop)
    constexpr int KS = KC / 4;
    static_assert(STAGES >= 3, "the consumer releases a stage one chunk late: needs >= 3 stages to overlap");
    int s = 0, s_prev = -1; uint32_t ph = 0;
    for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    int tn, tm; long long z;
    decode(tile, tm, tn, z);
    const int n0 = tn * BN, m0 = tm * BM;
    double cr[TM][TN][2], ci[TM][TN][2], cs[M3 ? TM : 1][M3 ? TN : 1][2];
#pragma unroll
    for (int i = 0; i < TM; ++i)
#pragma unroll
        for (int j = 0; j < TN; ++j) {
            cr[i][j][0] = cr[i][j][1] = 0.0; ci[i][j][0] = ci[i][j][1] = 0.0;
            if (M3) cs[i][j][0] = cs[i][j][1] = 0.0;
        }

    // Kpad is a multiple of KC (host contract): every chunk has KC/4 full k-steps, so the k-step loop is
    // straight-line code.  Fragments are double-buffered in registers: the LDS.128 of k-step k4+1 are issued
    // before the DMMAs of k-step k4, so their latency hides behind 3*TM*TN (or 4*TM*TN) tensor instructions.
    for (int c = 0; c < nchunks; ++c) {
        mbar_wait(full + s, ph);
        const double2* a_base = As + ((size_t)s * KC + t) * LDA + wm * TM * 8 + g;
        const double2* b_base = Bs + ((size_t)s * KC + t) * LDB + wn * TN * 8 + g;
        double2 a[2][TM], b[2][TN];
#pragma unroll
        for (int i = 0; i < TM; ++i) a[0][i] = a_base[i * 8];
#pragma unroll
        for (int j = 0; j < TN; ++j) b[0][j] = b_base[j * 8];
#pragma unroll
        for (int k4 = 0; k4 < KS; ++k4) {
            const int cur = k4 & 1, nxt = cur ^ 1;
            if (k4 + 1 < KS) {
#pragma unroll
                for (int i = 0; i < TM; ++i) a[nxt][i] = a_base[(size_t)(k4 + 1) * 4 * LDA + i * 8];
#pragma unroll
                for (int j = 0; j < TN; ++j) b[nxt][j] = b_base[(size_t)(k4 + 1) * 4 * LDB + j * 8];
            }
            if (M3) {
                double as[TM], bs[TN];
#pragma unroll
                for (int i = 0; i < TM; ++i) as[i] = a[cur][i].x + a[cur][i].y;
#pragma unroll
                for (int j = 0; j < TN; ++j) bs[j] = b[cur][j].x + b[cur][j].y;
#pragma unroll
                for (int i = 0; i < TM; ++i)
#pragma unroll
                    for (int j = 0; j < TN; ++j) {
                        dmma884(cr[i][j][0], cr[i][j][1], a[cur][i].x, b[cur][j].x);
                        dmma884(ci[i][j][0], ci[i][j][1], a[cur][i].y, b[cur][j].y);
                        dmma884(cs[i][j][0], cs[i][j][1], as[i], bs[j]);
                    }
            } else {
#pragma unroll
                for (int i = 0; i < TM; ++i) {
                    const double npi = neg(a[cur][i].y);
#pragma unroll
                    for (int j = 0; j < TN; ++j) {
                        dmma884(cr[i][j][0], cr[i][j][1], a[cur][i].x, b[cur][j].x);
                        dmma884(ci[i][j][0], ci[i][j][1], a[cur][i].x, b[cur][j].y);
                        dmma884(cr[i][j][0], cr[i][j][1], npi, b[cur][j].y);
                        dmma884(ci[i][j][0], ci[i][j][1], a[cur][i].y, b[cur][j].x);
                    }
                }
            }
        }
        // Release the PREVIOUS stage, not this one: ptxas schedules the arrive right behind the ISSUE of the last
        // LDS of the chunk (ahead of the DMMAs that consume them), and an LDS.128 still in flight then races with the
        // producer's next bulk copy into the stage (seen on B200 as wrong A fragments in the last quarter-warp when the
        // producer is starved and refills at once).  One chunk later every LDS of that stage has long been consumed.
        __syncwarp();
        if (lane == 0 && s_prev >= 0) mbar_arrive(empty + s_prev);
        s_prev = s;
        if (++s == STAGES) { s = 0; ph ^= 1u; }
    }
    if (M3) {
#pragma unroll
        for (int i = 0; i < TM; ++i)
#pragma unroll
            for (int j = 0; j < TN; ++j)
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const double t1 = cr[i][j][h], t2 = ci[i][j][h];
                    cr[i][j][h] = t1 - t2;
                    ci[i][j][h] = cs[i][j][h] - t1 - t2;
                }
    }

    // ---------------- store C (complex interleaved) ----------------
#pragma unroll
    for (int i = 0; i < TM; ++i) {
        const int mm = m0 + wm * TM * 8 + i * 8 + g;
        if (mm >= M) continue;
#pragma unroll
        for (int j = 0; j < TN; ++j) {
            const int n = n0 + wn * TN * 8 + j * 8 + 2 * t;
            double2* dst = C + (size_t)z * strideC + (size_t)mm * ldc;
            if (n < N) dst[cmap_off(n, cm)] = make_double2(cr[i][j][0], ci[i][j][0]);
            if (n + 1 < N) dst[cmap_off(n + 1, cm)] = make_double2(cr[i][j][1], ci[i][j][1]);
        }
    }
    }   // tile loop
}

// Standalone form of the same sum for the plain rotation path (nm > 48): one warp per (chunk of QC
// q-points, b1) reads the stored |g|^2 and writes partial[chunk][b1].
__global__ void __launch_bounds__(32)
k_rates_from_out(const double* __restrict__ outv /* [nq][nb1][nb2][nm] */, const double* __restrict__ omega, int nq,
                 int nm, int nb1, int nb2, int QC, RateArgs ra)
{
    const int b1 = blockIdx.y, qa = blockIdx.x * QC, qb = min(nq, qa + QC);
    const int per_q = nb2 * nm, lane = threadIdx.x;
    const double e1 = ra.eps_k[b1];
    double acc = 0.0;
    for (int i = lane; i < (qb - qa) * per_q; i += 32) {
        const int iq = qa + i / per_q, r = i % per_q, b2 = r / nm, nu = r - b2 * nm;
        const double w = omega[(size_t)iq * nm + nu];
        if (!(w > 0.0)) continue;
        const double e2 = ra.eps_kq[(size_t)iq * nb2 + b2];
        const double f2 = 1.0 / (exp((e2 - ra.mu) * ra.inv_kT) + 1.0), bn = 1.0 / (exp(w * ra.inv_kT) - 1.0);
        const double dm = e1 - w - e2, dp = e1 + w - e2;
        const double W = (1.0 - f2 + bn) * exp(-(dm * dm) * ra.inv_sigma2) + (f2 + bn) * exp(-(dp * dp) * ra.inv_sigma2);
        acc = fma(outv[(((size_t)iq * nb1 + b1) * nb2 + b2) * nm + nu], W, acc);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) ra.partial[(size_t)blockIdx.x * nb1 + b1] = acc;
}

// rate[b1] += scale * sum_j partial[j][b1], j in a fixed (strided, then tree) order: deterministic.
__global__ void __launch_bounds__(256)
k_rate_reduce(const double* __restrict__ partial, int nparts, int nb1, double scale, double* __restrict__ rate)
{
    // blockIdx.y = k slot of the stacked form (its own nparts rows of partial and its own rate[nb1]); 0 otherwise
    __shared__ double sh[256];
    const int b1 = blockIdx.x;
    partial += (size_t)blockIdx.y * nparts * nb1;
    rate += (size_t)blockIdx.y * nb1;
    double s = 0.0;
    for (int j = threadIdx.x; j < nparts; j += 256) s += partial[(size_t)j * nb1 + b1];
    sh[threadIdx.x] = s;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) rate[b1] += scale * sh[0];
}

// ---------------------------------------------------------------------------
// a5..a7: per (q, group of b1): rotate by conj(Ukq), by ev, square, scale.
// Plain shared-memory DFMA version: the fallback for nm > 48 (NT > 6).
// smem: Uc[nw][nb2] (already conjugated), Z[nm][nm], Cs[gb1][nw*nm], Ds[gb1][nb2*nm]
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_rotate_epilogue(const double2* __restrict__ C, long long ldc, int P, int PB, const double2* __restrict__ Ukq,
                  const double2* __restrict__ ev, const double* __restrict__ omega, double* __restrict__ out,
                  int nw, int nm, int nb1, int nb2, int gb1, PolarArgs pa)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double2* Uc = reinterpret_cast<double2*>(smem_raw);
    double2* Z = Uc + nw * nb2;
    double2* Cs = Z + nm * nm;
    double2* Ds = Cs + (size_t)gb1 * nw * nm;
    const int iq = blockIdx.y;
    const int b10 = blockIdx.x * gb1;
    const int nb1l = min(gb1, nb1 - b10);
    const int Y = nw * nm;
    const double2* Uq = Ukq + (size_t)iq * nw * nb2;
    for (int i = threadIdx.x; i < nw * nb2; i += blockDim.x) { double2 u = Uq[i]; Uc[i] = make_double2(u.x, (pa.conv & 1) ? u.y : -u.y); }
    const double2* Zq = ev + (size_t)iq * nm * nm;
    for (int i = threadIdx.x; i < nm * nm; i += blockDim.x) { double2 zv = Zq[i]; if (pa.conv & 2) zv.y = -zv.y; Z[i] = zv; }
    const double2* Cq = C + (size_t)iq * ldc + (size_t)b10 * PB;      // element (b1, w2, ka) at b1*PB + w2*P + ka
    for (int i = threadIdx.x; i < nb1l * Y; i += blockDim.x) {
        const int b1 = i / Y, r = i - b1 * Y, w2 = r / nm, ka = r - w2 * nm;
        Cs[i] = Cq[(size_t)b1 * PB + (size_t)w2 * P + ka];
    }
    __syncthreads();
    // a5
    const int nD = nb1l * nb2 * nm;
    for (int idx = threadIdx.x; idx < nD; idx += blockDim.x) {
        const int ka = idx % nm;
        const int b2 = (idx / nm) % nb2;
        const int b1 = idx / (nm * nb2);
        double sr = 0.0, si = 0.0;
        const double2* cc = Cs + (size_t)b1 * Y + ka;
        for (int w2 = 0; w2 < nw; ++w2) {
            const double2 u = Uc[w2 * nb2 + b2];
            const double2 c = cc[w2 * nm];
            sr = fma(u.x, c.x, sr); sr = fma(-u.y, c.y, sr);
            si = fma(u.x, c.y, si); si = fma(u.y, c.x, si);
        }
        Ds[idx] = make_double2(sr, si);
    }
    __syncthreads();
    // a6 + a7
    const double* om = omega + (size_t)iq * nm;
    double* o = out + ((size_t)iq * nb1 + b10) * nb2 * nm;
    for (int idx = threadIdx.x; idx < nD; idx += blockDim.x) {
        const int nu = idx % nm;
        const double2* d = Ds + (idx - nu);
        double sr = 0.0, si = 0.0;
        for (int ka = 0; ka < nm; ++ka) {
            const double2 z = Z[ka * nm + nu];
            const double2 c = d[ka];
            sr = fma(c.x, z.x, sr); sr = fma(-c.y, z.y, sr);
            si = fma(c.x, z.y, si); si = fma(c.y, z.x, si);
        }
        if (pa.P != nullptr) {          // f4: + P[q][nu] * [U_kq^dagger U_k]_{b2 b1}
            const int b2 = (idx / nm) % nb2, b1 = b10 + idx / (nm * nb2);
            double orr = 0.0, oi = 0.0;
            for (int w2 = 0; w2 < nw; ++w2) {
                const double2 u = Uc[w2 * nb2 + b2], k = pa.Uk[(size_t)w2 * nb1 + b1];
                orr = fma(u.x, k.x, orr); orr = fma(-u.y, k.y, orr);
                oi = fma(u.x, k.y, oi); oi = fma(u.y, k.x, oi);
            }
            const double2 pz = pa.P[(size_t)iq * nm + nu];
            sr += pz.x * orr - pz.y * oi;
            si += pz.x * oi + pz.y * orr;
        }
        const double w = om[nu];
        o[idx] = (w > 0.0) ? (sr * sr + si * si) / (2.0 * w) : 0.0;
    }
}

}  // namespace pe
