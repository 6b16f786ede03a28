// rotate_v3.cuh -- steps a5..a7 (Eq. 13 / Eq. 70 rotations, Eq. 7 |g|^2) as ONE persistent,
// warp-specialised kernel on the FP64 tensor cores.
//
//   a5  D[b2][(b1,ka)] = sum_w2 Uh[b2][w2] C[b1][w2][ka]     A = Uh = conj(Ukq)^T (8x4 per k-step), K = nw
//   a6  E[b2][nu]      = sum_ka D[b2][(b1,ka)] Z[ka][nu]      A = D straight from the a5 accumulators, K = nm
//   a7  out = |E|^2 / (2 omega)       (+ f2: Eq. 29 linewidth sums, + f4: Eq. 14-15 polar amplitude)
//
// One CTA per SM walks the q list.  A PRODUCER warp brings every input of the next q-points into shared-memory
// rings with TMA 1-D bulk copies -- the C panel as one copy, U_kq and ev row by row into padded rows (conflict-free
// fragment loads), 1/(2 omega) and the occupation factors of Eq. 29 computed by its own lanes -- while EIGHT CONSUMER
// warps do nothing but LDS.128 -> DMMA -> store: no staging pass, no index arithmetic per element, no per-CTA
// prologue (the previous form spent 20 % of its warp time there and 15 % waiting for its one TMA copy; small cells
// were issue-bound on the staging loops).  The arithmetic of an item is that of the second form (rotate_v2.cuh,
// removed): the N dimension of a5 is the packed index (b1, ka) in "pairs" of 4 ka, the DMMA accumulators of a5 ARE
// the A fragments of a6, both products use the three-multiply complex product.  Conjugations are signs in the
// operand sums (conj(U): as = ur - ui, T2 enters with the opposite sign), so the raw inputs are used as they land.
//
// Two rings: the Q ring (U_kq, ev, 1/(2 omega), Eq. 29 factors of QS q-points per stage) and the C ring (the C panels
// of those q-points; for cells whose panel does not fit, groups of gb1 values of b1), three stages each.
//
// C layout (written by the contraction kernels): element (b1, w2, ka) of a q at b1*PB + w2*P + ka.  P = nm except
// for nm = 0 mod 4, where the row pitch is nm + 1: the four k rows (w2) of a B fragment then fall into distinct
// 16-byte bank groups.  For nm = 2 mod 4 the same is reached without padding by interleaving the two pairs of a
// column tile (ka = 8i + 2t' + h instead of 4s + t'): the order of the ka sum is free.
#pragma once
#include "ptx_helpers.cuh"
#include "rot_args.cuh"

namespace pe {

// Warpgroups of consumer warps plus one that holds the producer warp (its other three warps exit at once); the
// register file is re-split between them at kernel start (setmaxnreg).  Items with two tiles of b2 (MTW = 2) need
// ~230 registers: 8 consumer warps (8 x 232 + 4 x 40 = 12 x 168); items with one tile fit 160: 12 consumer warps
// (12 x 160 + 4 x 32 = 16 x 128), three per scheduler -- more warps to overlap one item's DMMA phases with another's
// operand sums / epilogue.
#ifndef PHOEBE_ROT3_NCW1
#define PHOEBE_ROT3_NCW1 12
#endif
__host__ __device__ constexpr int rot3_consumers(int MTW) { return MTW == 2 ? 8 : PHOEBE_ROT3_NCW1; }
__host__ __device__ constexpr int rot3_threads(int MTW) { return (rot3_consumers(MTW) + 4) * 32; }
constexpr int kRot3Stages = 3;

struct Rot3Layout {
    int KS, NT, MT, nwp, ldu, ldz, mapB, slack;
    uint32_t szU, szZ, szW, szR, szQ, szC, off_Q, off_C, total;      // bytes
};

// row pitch of the C layout for nm modes, and the b1 block pitch (pad chosen by the host, see rot3_block_pad)
__host__ __device__ inline int rot3_row_pitch(int nm) { return (nm & 3) == 0 ? nm + 1 : nm; }

// blk: U_kq / ev of a q-point land as ONE bulk copy each, rows at their natural pitch (small cells: a bulk copy per
// 64..128-byte row costs the TMA unit more than the few bank conflicts of the unpadded rows cost the consumers);
// otherwise row by row into padded rows.
__host__ __device__ inline Rot3Layout rot3_layout(int nw, int nm, int nb2, int PB, int QS, int gb1, bool rates, bool blk)
{
    Rot3Layout L;
    const int P = rot3_row_pitch(nm);
    L.KS = (nm + 3) >> 2; L.NT = (nm + 7) >> 3; L.MT = (nb2 + 7) >> 3;
    L.nwp = (nw + 3) & ~3;
    L.mapB = (nm & 3) == 2;
    L.ldu = blk ? nb2 : L.MT * 8 + 2;           // complex; = 2 mod 8: the 4 k rows of an A fragment hit distinct bank groups
    L.ldz = blk ? nm : L.NT * 8 + (L.mapB ? 1 : 2);    // mapB reads rows 2t apart: an odd pitch spreads them
    L.slack = 3 * P + 4 * L.KS + 4;             // what the padded k rows / columns behind the last panel may read
    // (blk: the last rows' column padding reads up to 7 elements past a q-point's block)
    L.szU = (uint32_t)(QS * L.nwp * L.ldu + (blk ? 8 : 0)) * 16;
    L.szZ = (uint32_t)(QS * 4 * L.KS * L.ldz + (blk ? 8 : 0)) * 16;
    L.szW = (uint32_t)QS * 8 * L.NT * 8;
    L.szR = rates ? (uint32_t)QS * (2 * 8 * L.NT + 2 * 8 * L.MT) * 8 : 0u;
    L.szQ = L.szU + L.szZ + L.szW + L.szR;
    L.szC = (uint32_t)(QS * gb1 * PB + L.slack) * 16;
    L.off_Q = 128;                              // 4 x kRot3Stages mbarriers in front
    L.off_C = L.off_Q + kRot3Stages * L.szQ;
    L.total = L.off_C + kRot3Stages * L.szC;
    return L;
}

struct Rot3Args {
    const double2* C;       // [nq][nb1*PB]
    const double2* Ukq;     // [nq][nw][nb2]
    const double2* ev;      // [nq][nm][nm]
    const double* omega;    // [nq][nm]
    double* out;            // [nq][nb1][nb2][nm] or nullptr (RATES only)
    int nq, nw, nm, nb1, nb2;
    int PB, QS, gb1;
    int blk;                // U_kq / ev as one block per q-point (rot3_layout)
    RateArgs ra;            // ra.partial: [nq][nmg][nb1]
    PolarArgs pa;
};

// ka covered by lane t' of pair s (the order of the ka sum of a6 is free; both a5's B columns and a6's Z rows use it)
template <int KS>
__device__ __forceinline__ int rot3_kappa(int s, int tt, int mapB)
{
    if (mapB && s < (KS & ~1)) return 8 * (s >> 1) + (s & 1) + 2 * tt;
    return 4 * s + tt;
}

// MODE: 0 = |g|^2 only, 1 = with the linewidth sums of Eq. 29 (f2), 3 = with the polar term of Eq. 14-15 (f4; the
// linewidth sums are then a run-time choice: a.ra.eps_k != nullptr)
template <int KS, int GB, int MTW, int MODE>
__global__ void __launch_bounds__(rot3_threads(MTW), 1)
k_rotate_v3(const Rot3Args a)
{
    constexpr int NCW = rot3_consumers(MTW), NTHREADS = rot3_threads(MTW);
    constexpr int REGS_C = MTW == 2 ? 232 : (NCW == 16 ? 112 : 160), REGS_P = MTW == 2 ? 40 : 32;
    constexpr bool RSM = (MODE & 1) != 0;                 // the Eq. 29 arrays exist in the Q stages
    constexpr bool POLAR = (MODE & 2) != 0;
    const bool rates = RSM && (MODE != 3 || a.ra.eps_k != nullptr);
    constexpr int TJ = (GB * KS + 1) / 2;                 // a5 column tiles per item
    constexpr int NT = (KS + 1) / 2;
    constexpr int NS = kRot3Stages;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int nw = a.nw, nm = a.nm, nb1 = a.nb1, nb2 = a.nb2, PB = a.PB, QS = a.QS, gb1 = a.gb1;
    const int P = rot3_row_pitch(nm);
    const Rot3Layout L = rot3_layout(nw, nm, nb2, PB, QS, gb1, RSM, a.blk != 0);
    const int MT = L.MT, ldu = L.ldu, ldz = L.ldz, nwp = L.nwp, mapB = L.mapB;
    const int ngroups = (nb1 + gb1 - 1) / gb1;
    uint64_t* qfull = reinterpret_cast<uint64_t*>(smem_raw);
    uint64_t* qempty = qfull + NS;
    uint64_t* cfull = qempty + NS;
    uint64_t* cempty = cfull + NS;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    // the rings are zeroed ONCE: the bulk copies only ever write the real rows / columns, so the padding the fragment
    // loads touch (U rows >= nw, Z rows >= nm, row tails, the slack behind the panels) stays zero for the whole kernel
    for (uint32_t i = L.off_Q / 16 + threadIdx.x; i < L.total / 16; i += NTHREADS)
        reinterpret_cast<double2*>(smem_raw)[i] = make_double2(0.0, 0.0);
    // Warp w takes the items w, w + NCW, ... of the CTA's whole item SEQUENCE (not of each stage), so a stage with
    // fewer items than warps does not leave the same warps idle every time, and the warps drift apart across the
    // stages of the ring instead of marching through them in step.  Every warp observes every stage (waits for its
    // full barrier, arrives on its empty barrier) in order, with or without items in it: barrier phases stay in step.
    if (threadIdx.x == 0) {
        for (int s = 0; s < NS; ++s) {
            mbar_init(qfull + s, 1); mbar_init(qempty + s, NCW);
            mbar_init(cfull + s, 1); mbar_init(cempty + s, NCW);
        }
        mbar_fence_init();
    }
    fence_proxy_async();
    __syncthreads();

    const int nqg = (a.nq + QS - 1) / QS;
    const long long ldcq = (long long)nb1 * PB;

    if (warp >= NCW) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(REGS_P));
        if (warp > NCW) return;
        // ================= producer warp =================
        int sq = 0, sc = 0; uint32_t phq = 0, phc = 0;
        const int nW = 8 * NT, nE = 8 * MT;
        for (int qg = blockIdx.x; qg < nqg; qg += gridDim.x) {
            const int q0 = qg * QS, nql = min(QS, a.nq - q0);
            // omega (and eps_kq) of this stage: loads issued BEFORE the wait for a free stage
            constexpr int WR = 4;                            // register slots per lane (QS * 8NT <= 32 * WR by host contract)
            double wv[WR], ev2[RSM ? WR : 1];
#pragma unroll
            for (int r = 0; r < WR; ++r) {
                const int i = lane + 32 * r, ql = i / nW, nu = i - ql * nW;
                wv[r] = (ql < nql && nu < nm) ? a.omega[(size_t)(q0 + ql) * nm + nu] : 0.0;
                if (RSM) {
                    const int qe = i / nE, b2 = i - qe * nE;
                    ev2[r] = (rates && qe < nql && b2 < nb2) ? a.ra.eps_kq[(size_t)(q0 + qe) * nb2 + b2] : 0.0;
                }
            }
            mbar_wait(qempty + sq, phq ^ 1u);
            unsigned char* Q = smem_raw + L.off_Q + (size_t)sq * L.szQ;
            double2* Us = reinterpret_cast<double2*>(Q);
            double2* Zs = reinterpret_cast<double2*>(Q + L.szU);
            double* iw = reinterpret_cast<double*>(Q + L.szU + L.szZ);
            if (a.blk) {
                // one copy per q-point (all q-points at once when there are no padding rows between their blocks)
                if (nwp == nw) {
                    if (lane == 0) bulk_g2s(Us, a.Ukq + (size_t)q0 * nw * nb2, (uint32_t)(nql * nw * nb2) * 16u, qfull + sq);
                } else if (lane < nql) {
                    bulk_g2s(Us + (size_t)lane * nwp * ldu, a.Ukq + (size_t)(q0 + lane) * nw * nb2, (uint32_t)(nw * nb2) * 16u,
                             qfull + sq);
                }
                if (4 * KS == nm) {
                    if (lane == 1) bulk_g2s(Zs, a.ev + (size_t)q0 * nm * nm, (uint32_t)(nql * nm * nm) * 16u, qfull + sq);
                } else if (lane < nql) {
                    bulk_g2s(Zs + (size_t)lane * 4 * KS * ldz, a.ev + (size_t)(q0 + lane) * nm * nm, (uint32_t)(nm * nm) * 16u,
                             qfull + sq);
                }
            } else {
                for (int i = lane; i < nql * nw; i += 32) {          // U_kq rows: [q][w2][nb2] -> Us[ql][w2][ldu]
                    const int ql = i / nw, w2 = i - ql * nw;
                    bulk_g2s(Us + ((size_t)ql * nwp + w2) * ldu, a.Ukq + ((size_t)(q0 + ql) * nw + w2) * nb2,
                             (uint32_t)nb2 * 16u, qfull + sq);
                }
                for (int i = lane; i < nql * nm; i += 32) {          // ev rows: [q][ka][nm] -> Zs[ql][ka][ldz]
                    const int ql = i / nm, ka = i - ql * nm;
                    bulk_g2s(Zs + ((size_t)ql * 4 * KS + ka) * ldz, a.ev + ((size_t)(q0 + ql) * nm + ka) * nm,
                             (uint32_t)nm * 16u, qfull + sq);
                }
            }
#pragma unroll
            for (int r = 0; r < WR; ++r) {
                const int i = lane + 32 * r;
                if (i < QS * nW) iw[i] = (wv[r] > 0.0) ? 0.5 / wv[r] : 0.0;
                if (RSM) {
                    double* om_s = iw + QS * nW;
                    double* bose_s = om_s + QS * nW;
                    double* e2_s = bose_s + QS * nW;
                    double* f2_s = e2_s + QS * nE;
                    if (i < QS * nW) {
                        om_s[i] = wv[r];
                        bose_s[i] = (wv[r] > 0.0) ? 1.0 / (exp(wv[r] * a.ra.inv_kT) - 1.0) : 0.0;
                    }
                    if (i < QS * nE) {
                        const int qe = i / nE, b2 = i - qe * nE;
                        e2_s[i] = ev2[r];
                        f2_s[i] = (qe < nql && b2 < nb2) ? 1.0 / (exp((ev2[r] - a.ra.mu) * a.ra.inv_kT) + 1.0) : 0.0;
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive_expect_tx(qfull + sq, (uint32_t)nql * (uint32_t)(nw * nb2 + nm * nm) * 16u);
            if (++sq == NS) { sq = 0; phq ^= 1u; }
            for (int grp = 0; grp < ngroups; ++grp) {
                mbar_wait(cempty + sc, phc ^ 1u);
                if (lane == 0) {
                    const int b10 = grp * gb1, nb1l = min(gb1, nb1 - b10);
                    // whole q-points (ngroups == 1): the panels of the nql q-points are contiguous in C
                    const uint32_t bytes = (uint32_t)(ngroups == 1 ? (long long)nql * ldcq : (long long)nb1l * PB) * 16u;
                    mbar_arrive_expect_tx(cfull + sc, bytes);
                    bulk_g2s(smem_raw + L.off_C + (size_t)sc * L.szC, a.C + (size_t)q0 * ldcq + (size_t)b10 * PB, bytes,
                             cfull + sc);
                }
                if (++sc == NS) { sc = 0; phc ^= 1u; }
            }
        }
        return;
    }

    // ================= consumer warps =================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(REGS_C));
    const int g = lane >> 2, t = lane & 3;
    const double nsU = (a.pa.conv & 1) ? -1.0 : 1.0;      // MINUS the sign Im U enters with (default: conjugated)
    const double nsZ = (a.pa.conv & 2) ? 1.0 : -1.0;      // MINUS the sign Im Z enters with (default: plain)
    const int nks = nwp >> 2;
    int zrow[KS];                                        // Z row (times its pitch) of this lane in k-step s of a6
#pragma unroll
    for (int s = 0; s < KS; ++s) zrow[s] = rot3_kappa<KS>(s, t, mapB) * ldz + g;
    const int nmg = (MT + MTW - 1) / MTW;
    const int so_b1 = nb2 * nm, so_mt = 8 * nm;          // strides of out in b1 and in tiles of b2
    // this lane's B column of a5 tile j: which b1 of the item (cbl) and where in the C panel (cof, without the b1 term)
    int cbl[TJ], cof[TJ];
#pragma unroll
    for (int j = 0; j < TJ; ++j) {
        const int p = min(2 * j + (g & 1), GB * KS - 1);        // pair of the column (clamped: unused half tile)
        const int bl = p / KS, sp = p - bl * KS;
        cbl[j] = bl;
        cof[j] = t * P + rot3_kappa<KS>(sp, g >> 1, mapB);
    }
    const int uof = t * ldu + g;                         // A fragment of a5: row t of a k-step, column g of a tile of b2
    // two consecutive outputs of a lane are one aligned 16-byte store
    const bool st2 = (nm & 1) == 0 && (reinterpret_cast<uintptr_t>(a.out) & 15u) == 0;
    int sq = 0, sc = 0; uint32_t phq = 0, phc = 0;       // slot and phase parity of the two rings
    int rem = 0;                     // (items of all earlier stages) % NCW
    const int nbg_full = (min(gb1, nb1) + GB - 1) / GB;
    for (int qg = blockIdx.x; qg < nqg; qg += gridDim.x) {
        const int q0 = qg * QS, nql = min(QS, a.nq - q0);
        mbar_wait(qfull + sq, phq);
        const unsigned char* Q = smem_raw + L.off_Q + (size_t)sq * L.szQ;
        const double2* Us = reinterpret_cast<const double2*>(Q);
        const double2* Zs = reinterpret_cast<const double2*>(Q + L.szU);
        const double* iwq = reinterpret_cast<const double*>(Q + L.szU + L.szZ);
        const double* om_s = iwq + QS * 8 * NT;
        const double* bose_s = om_s + QS * 8 * NT;
        const double* e2_s = bose_s + QS * 8 * NT;
        const double* f2_s = e2_s + QS * 8 * MT;
        for (int grp = 0; grp < ngroups; ++grp) {
            const double2* Cs = reinterpret_cast<const double2*>(smem_raw + L.off_C + (size_t)sc * L.szC);
            const int b10 = grp * gb1;
            const int nb1l = min(gb1, nb1 - b10);
            const int nbg = nb1l == gb1 ? nbg_full : (nb1l + GB - 1) / GB;
            const int per_q = nbg * nmg;
            const int ni = nql * per_q;
            int item = warp - rem; if (item < 0) item += NCW;           // this warp's first item of the stage
            rem = (rem + ni) % NCW;
            mbar_wait(cfull + sc, phc);
            for (; item < ni; item += NCW) {
                int ql = 0, r = item;
                if (nql > 1) { ql = (int)((unsigned)item / (unsigned)per_q); r = item - ql * per_q; }
                int bg = r, mg = 0;
                if (nmg > 1) { bg = (int)((unsigned)r / (unsigned)nmg); mg = r - bg * nmg; }
                const int b1a = bg * GB, mt0 = mg * MTW;
                // ---- a5: T1, T2, T3 of D[b2][(b1,ka)] ----
                double t1[MTW][TJ][2], t2[MTW][TJ][2], t3[MTW][TJ][2];
#pragma unroll
                for (int mi = 0; mi < MTW; ++mi)
#pragma unroll
                    for (int j = 0; j < TJ; ++j) {
                        t1[mi][j][0] = t1[mi][j][1] = 0.0; t2[mi][j][0] = t2[mi][j][1] = 0.0; t3[mi][j][0] = t3[mi][j][1] = 0.0;
                    }
                // running fragment pointers (one add per k-step each)
                const double2* ua[MTW];
#pragma unroll
                for (int mi = 0; mi < MTW; ++mi)
                    ua[mi] = Us + ql * (nwp * ldu) + uof + min(mt0 + mi, MT - 1) * 8;
                const double2* pbase = Cs + ql * (gb1 * PB);
                const double2* cb[TJ];
#pragma unroll
                for (int j = 0; j < TJ; ++j) cb[j] = pbase + min(b1a + cbl[j], nb1l - 1) * PB + cof[j];
                // f4: the overlap O[b2][b1] = sum_w Uh[b2][w] Uk[w][b1] as one more column tile per two b1 (columns
                // alternate between the two b1, so every lane ends up with O of both in its accumulator pair)
                constexpr int TO = POLAR ? (GB + 1) / 2 : 1;
                double o1[MTW][TO][2], o2[MTW][TO][2], o3[MTW][TO][2];
                const double2* kb[TO];
                if (POLAR) {
#pragma unroll
                    for (int mi = 0; mi < MTW; ++mi)
#pragma unroll
                        for (int jo = 0; jo < TO; ++jo) {
                            o1[mi][jo][0] = o1[mi][jo][1] = 0.0; o2[mi][jo][0] = o2[mi][jo][1] = 0.0; o3[mi][jo][0] = o3[mi][jo][1] = 0.0;
                        }
#pragma unroll
                    for (int jo = 0; jo < TO; ++jo) kb[jo] = a.pa.Uk + min(b10 + b1a + 2 * jo + (g & 1), nb1 - 1);
                }
                // one k-step (4 values of w2): fragments (av, bv) are consumed, those of the next step land in (an, bn)
                auto kstep = [&](const double2 (&av)[MTW], const double2 (&bv)[TJ], double2 (&an)[MTW], double2 (&bn)[TJ],
                                 int ks, bool more) {
                    double as[MTW], bs[TJ];
#pragma unroll
                    for (int mi = 0; mi < MTW; ++mi) as[mi] = fma(-nsU, av[mi].y, av[mi].x);
#pragma unroll
                    for (int j = 0; j < TJ; ++j) bs[j] = bv[j].x + bv[j].y;
                    if (more) {
#pragma unroll
                        for (int mi = 0; mi < MTW; ++mi) { ua[mi] += 4 * ldu; an[mi] = *ua[mi]; }
#pragma unroll
                        for (int j = 0; j < TJ; ++j) { cb[j] += 4 * P; bn[j] = *cb[j]; }
                    }
#pragma unroll
                    for (int mi = 0; mi < MTW; ++mi)
#pragma unroll
                        for (int j = 0; j < TJ; ++j) {
                            dmma884(t1[mi][j][0], t1[mi][j][1], av[mi].x, bv[j].x);
                            dmma884(t2[mi][j][0], t2[mi][j][1], av[mi].y, bv[j].y);
                            dmma884(t3[mi][j][0], t3[mi][j][1], as[mi], bs[j]);
                        }
                    if (POLAR) {
#pragma unroll
                        for (int jo = 0; jo < TO; ++jo) {
                            const double2 kv = kb[jo][(size_t)min(4 * ks + t, nw - 1) * nb1];
                            const double ksum = kv.x + kv.y;
#pragma unroll
                            for (int mi = 0; mi < MTW; ++mi) {
                                dmma884(o1[mi][jo][0], o1[mi][jo][1], av[mi].x, kv.x);
                                dmma884(o2[mi][jo][0], o2[mi][jo][1], av[mi].y, kv.y);
                                dmma884(o3[mi][jo][0], o3[mi][jo][1], as[mi], ksum);
                            }
                        }
                    }
                };
                {
                    double2 fa0[MTW], fb0[TJ], fa1[MTW], fb1[TJ];      // two fragment sets used alternately: no register moves
#pragma unroll
                    for (int mi = 0; mi < MTW; ++mi) fa0[mi] = *ua[mi];
#pragma unroll
                    for (int j = 0; j < TJ; ++j) fb0[j] = *cb[j];
                    for (int ks = 0; ks < nks; ks += 2) {
                        kstep(fa0, fb0, fa1, fb1, ks, ks + 1 < nks);
                        if (ks + 1 < nks) kstep(fa1, fb1, fa0, fb0, ks + 1, ks + 2 < nks);
                    }
                }
                // D = (T1 -+ T2) + i (T3 - T1 -+ T2); kept as (Re, Im, Re + Im): the three A planes of a6
#pragma unroll
                for (int mi = 0; mi < MTW; ++mi)
#pragma unroll
                    for (int j = 0; j < TJ; ++j)
#pragma unroll
                        for (int h = 0; h < 2; ++h) {
                            const double x1 = t1[mi][j][h], x2 = t2[mi][j][h], x3 = t3[mi][j][h];
                            const double re = fma(nsU, x2, x1), im = fma(nsU, x2, x3 - x1);
                            t1[mi][j][h] = re; t2[mi][j][h] = im; t3[mi][j][h] = re + im;
                        }
                if (POLAR) {
#pragma unroll
                    for (int mi = 0; mi < MTW; ++mi)
#pragma unroll
                        for (int jo = 0; jo < TO; ++jo)
#pragma unroll
                            for (int h = 0; h < 2; ++h) {
                                const double x1 = o1[mi][jo][h], x2 = o2[mi][jo][h], x3 = o3[mi][jo][h];
                                o1[mi][jo][h] = fma(nsU, x2, x1); o2[mi][jo][h] = fma(nsU, x2, x3 - x1);
                            }
                }
                // ---- a6 + a7 ----
                const double2* zq = Zs + (size_t)ql * 4 * KS * ldz;
                const double* iw = iwq + ql * 8 * NT;
                const int qabs = q0 + ql;
                double racc[GB], e1k[GB];
                bool okb[GB], okm[MTW];
#pragma unroll
                for (int bl = 0; bl < GB; ++bl) {
                    racc[bl] = 0.0;
                    okb[bl] = b1a + bl < nb1l;
                    e1k[bl] = rates ? a.ra.eps_k[(a.ra.rows_per_k > 0 ? (qabs / a.ra.rows_per_k) * nb1 : 0) +
                                                 min(b10 + b1a + bl, nb1 - 1)] : 0.0;
                }
#pragma unroll
                for (int mi = 0; mi < MTW; ++mi) okm[mi] = mt0 + mi < MT && (mt0 + mi) * 8 + g < nb2;
                // out[q][b1][b2][nu] of this lane's first value; + bl * so_b1 + mi * so_mt + 8 n for the others
                double* obase = a.out + (((size_t)qabs * nb1 + b10 + b1a) * nb2 + (size_t)mt0 * 8 + g) * nm + 2 * t;
#pragma unroll 1
                for (int n = 0; n < NT; ++n) {
                    double e1[GB][MTW][2], e2[GB][MTW][2], e3[GB][MTW][2];
#pragma unroll
                    for (int bl = 0; bl < GB; ++bl)
#pragma unroll
                        for (int mi = 0; mi < MTW; ++mi) {
                            e1[bl][mi][0] = e1[bl][mi][1] = 0.0; e2[bl][mi][0] = e2[bl][mi][1] = 0.0; e3[bl][mi][0] = e3[bl][mi][1] = 0.0;
                        }
#pragma unroll
                    for (int s = 0; s < KS; ++s) {
                        const double2 z = zq[zrow[s] + 8 * n];
                        const double zs = fma(-nsZ, z.y, z.x);
#pragma unroll
                        for (int bl = 0; bl < GB; ++bl) {
                            const int p = bl * KS + s, j = p >> 1, h = p & 1;
#pragma unroll
                            for (int mi = 0; mi < MTW; ++mi) {
                                dmma884(e1[bl][mi][0], e1[bl][mi][1], t1[mi][j][h], z.x);
                                dmma884(e2[bl][mi][0], e2[bl][mi][1], t2[mi][j][h], z.y);
                                dmma884(e3[bl][mi][0], e3[bl][mi][1], t3[mi][j][h], zs);
                            }
                        }
                    }
                    // branch-free: every lane computes its two values, only the stores are predicated
                    const int nu = 8 * n + 2 * t;
                    const double2 iw2 = *reinterpret_cast<const double2*>(iw + nu);      // 1/(2 omega) of this lane's two columns
                    const bool ok0 = nu < nm, ok1 = nu + 1 < nm;
                    double2 pz[2] = {make_double2(0.0, 0.0), make_double2(0.0, 0.0)};
                    if (POLAR) {
                        if (ok0) pz[0] = a.pa.P[(size_t)qabs * nm + nu];
                        if (ok1) pz[1] = a.pa.P[(size_t)qabs * nm + nu + 1];
                    }
#pragma unroll
                    for (int bl = 0; bl < GB; ++bl) {
#pragma unroll
                        for (int mi = 0; mi < MTW; ++mi) {
                            const bool okr = okb[bl] && okm[mi];            // this lane's (b1, b2) exists
                            double er[2], ei[2];
#pragma unroll
                            for (int h = 0; h < 2; ++h) {
                                er[h] = fma(nsZ, e2[bl][mi][h], e1[bl][mi][h]);
                                ei[h] = fma(nsZ, e2[bl][mi][h], e3[bl][mi][h] - e1[bl][mi][h]);
                            }
                            if (POLAR) {
                                const double ox = o1[mi][bl >> 1][bl & 1], oy = o2[mi][bl >> 1][bl & 1];
#pragma unroll
                                for (int h = 0; h < 2; ++h) {
                                    er[h] += pz[h].x * ox - pz[h].y * oy;
                                    ei[h] += pz[h].x * oy + pz[h].y * ox;
                                }
                            }
                            const double v0 = (er[0] * er[0] + ei[0] * ei[0]) * iw2.x;
                            const double v1 = (er[1] * er[1] + ei[1] * ei[1]) * iw2.y;
                            if (!RSM || a.out != nullptr) {
                                double* orow = obase + (size_t)bl * so_b1 + (size_t)mi * so_mt + 8 * n;
                                if (st2) { if (okr && ok1) *reinterpret_cast<double2*>(orow) = make_double2(v0, v1); }
                                else { if (okr && ok0) orow[0] = v0; if (okr && ok1) orow[1] = v1; }
                                if (st2 && okr && ok0 && !ok1) orow[0] = v0;
                            }
                            if (rates) {
                                const int b2c = min((mt0 + mi) * 8 + g, 8 * MT - 1);
                                const double x12 = e1k[bl] - e2_s[ql * 8 * MT + b2c];
                                const double f2 = f2_s[ql * 8 * MT + b2c];
#pragma unroll
                                for (int h = 0; h < 2; ++h) {
                                    const double w = om_s[ql * 8 * NT + nu + h], bn_ = bose_s[ql * 8 * NT + nu + h];
                                    const double dm = x12 - w, dp = x12 + w;
                                    const double W = (1.0 - f2 + bn_) * exp(-(dm * dm) * a.ra.inv_sigma2) +
                                                     (f2 + bn_) * exp(-(dp * dp) * a.ra.inv_sigma2);
                                    // padded rows / columns: omega = 0 there gives v = 0 exactly (1/(2 omega) := 0), rows
                                    // b2 >= nb2 are masked
                                    racc[bl] = fma((okr && (h ? ok1 : ok0)) ? (h ? v1 : v0) : 0.0, W, racc[bl]);
                                }
                            }
                        }
                    }
                }
                if (rates) {        // fixed-order sum over the warp: partial[q][mg][b1] is owned by this item
#pragma unroll
                    for (int bl = 0; bl < GB; ++bl) {
                        double rsum = racc[bl];
#pragma unroll
                        for (int o = 16; o > 0; o >>= 1) rsum += __shfl_xor_sync(0xffffffffu, rsum, o);
                        if (lane == 0 && b1a + bl < nb1l)
                            a.ra.partial[((size_t)qabs * nmg + mg) * nb1 + b10 + b1a + bl] = rsum;
                    }
                }
            }
            // Release the stage: every shared-memory load of an item has been consumed by the time its last store
            // issues (the stores depend on all of its DMMAs, those on all of its fragment loads); the fence keeps the
            // arrive behind those stores and orders every lane's reads before lane 0's release.
            __threadfence_block();
            __syncwarp();
            if (lane == 0) mbar_arrive(cempty + sc);
            if (++sc == NS) { sc = 0; phc ^= 1u; }
        }
        __threadfence_block();
        __syncwarp();
        if (lane == 0) mbar_arrive(qempty + sq);
        if (++sq == NS) { sq = 0; phq ^= 1u; }
    }
}

}  // namespace pe
