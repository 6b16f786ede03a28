// rotate_v2.cuh -- steps a5..a7 (Eq. 13 / Eq. 70 rotations, Eq. 7 |g|^2) on the FP64 tensor cores,
// second form: no padded k-steps in a6, three-multiply complex product in a5 and a6.
//
//   a5  D[b2][(b1,ka)] = sum_w2 Uh[b2][w2] C[b1][w2][ka]     A = Uh = conj(Ukq)^T (8x4 per k-step), K = nw
//   a6  E[b2][nu]      = sum_ka D[b2][(b1,ka)] Z[ka][nu]      A = D straight from the a5 accumulators, K = nm
//   a7  out = |E|^2 / (2 omega)
//
// What differs from k_rotate_epilogue_mma (qbatch_kernels.cuh):
//  * The N dimension of a5 is the PACKED index (b1, ka): the 8 columns of an a5 tile are two "pairs"
//    (b1, s), each covering ka = 4s .. 4s+3.  The DMMA accumulator of lane (g,t) holds columns 2t and 2t+1;
//    column 2t'+h of tile j is DEFINED to be ka = 4 s(j,h) + t' of pair 2j+h, so register h of tile j IS the
//    A fragment A[g][k = t] of a6's k-step s for that b1 -- no shuffles, no shared-memory round trip, and
//    a6 runs ceil(nm/4) k-steps instead of 2*ceil(nm/8) (nm = 12: 3 instead of 4; the padded half of the
//    last a5 tile is gone too).  Pairs per b1: KS = ceil(nm/4).  A warp item covers G b1 (G = 2 for KS = 1, 3
//    so that the pairs fill whole tiles) x MTW m-tiles of b2.
//  * Both products use the three-multiply complex product: T1 = sum ar*br, T2 = sum ai*bi,
//    T3 = sum (ar+ai)(br+bi); Re = T1 - T2, Im = T3 - T1 - T2.  3 DMMA per complex tile and k-step instead
//    of 4; the operand sums are one DADD per fragment (A of a5, B of a5), the a5 results (one DADD per
//    accumulator, once) and a precomputed third plane of Z.
//  * A B fragment of a5 feeds MTW m-tiles and a Z fragment of a6 feeds G*MTW tiles (v1: one each).
// Shared memory: as v1 (Us conj'd and zero padded, Zs zero padded, C panels by TMA bulk copy, zeroed
// slack) plus Zsum = Re Z + Im Z.  Reads of padded rows / columns hit finite values (zeroed slack, the
// next row of the panel) and multiply zero rows of Us / Zs.
#pragma once
#include "ptx_helpers.cuh"
#include "qbatch_kernels.cuh"

#ifndef PHOEBE_ROT_EB
#define PHOEBE_ROT_EB 3
#endif

namespace pe {

struct Rot2Layout {
    int KS, NT, MT, nwp, ldu, ldz, ldzs, slack, nbuf, ngroups;
    size_t panel;                                   // complex elements of one (q, group) buffer
    size_t off_inv2w, off_Us, off_Zs, off_Zsum, off_Cs, off_rates, off_polar, total;    // bytes
};

__host__ __device__ inline Rot2Layout rot2_layout(int QG, int nw, int nm, int nb1, int nb2, int gb1, bool rates, bool polar)
{
    Rot2Layout L;
    L.KS = (nm + 3) >> 2; L.NT = (nm + 7) >> 3; L.MT = (nb2 + 7) >> 3;
    L.nwp = (nw + 3) & ~3;
    L.ldu = L.MT * 8 + 2;                // complex; = 2 mod 8: A loads of a quarter-warp hit 8 distinct 16-B banks
    L.ldz = L.NT * 8 + 2;                // complex; rows 4s+t, columns 8n+g
    L.ldzs = L.NT * 8 + 4;               // doubles; = 4 or 12 mod 16: LDS.64 of a half-warp conflict-free
    L.slack = 4 * nm + 8;
    L.panel = (size_t)gb1 * nw * nm + L.slack;
    L.ngroups = (nb1 + gb1 - 1) / gb1;
    L.nbuf = L.ngroups > 1 ? 2 : 1;
    size_t o = 16;                                                     // two mbarriers
    L.off_inv2w = o; o += (size_t)QG * 8 * L.NT * 8;
    L.off_Us = o;    o += (size_t)QG * L.nwp * L.ldu * 16;
    L.off_Zs = o;    o += (size_t)QG * 4 * L.KS * L.ldz * 16;
    L.off_Zsum = o;  o += (size_t)QG * 4 * L.KS * L.ldzs * 8;
    L.off_Cs = o;    o += (size_t)L.nbuf * QG * L.panel * 16;
    L.off_rates = o;
    if (rates) o += ((size_t)QG * (2 * 8 * L.NT + 2 * 8 * L.MT) + (((size_t)4 * nb1 + 1) & ~(size_t)1)) * 8;
    L.off_polar = o;
    if (polar) o += ((size_t)QG * 8 * L.NT + (size_t)QG * nb1 * 8 * L.MT) * 16;
    L.total = o;
    return L;
}

// Second launch-bound argument (resident CTAs the register allocation must leave room for): 2 for the mid-size
// accumulator sets -- the large cell's two-m-tile variant gains from it (31.5 -> 29.7 ms); 0 (= unspecified) elsewhere:
// any tighter bound changes ptxas' schedule of the small-cell variants for the worse (band-window 2.50 -> 2.71 ms even at
// the same occupancy); 3 for the 4-atom variant, which sits on that register edge (168): at 2 CTAs its launch takes 6.3 ms
// instead of 3.8 ms.
template <int KS, int MTW, bool RATES>
__global__ void __launch_bounds__(128, (KS >= 5 && KS <= 8) ? 2 : ((KS == 3 || KS == 4) && MTW == 2 && !RATES) ? 3 : 0)
k_rotate_epilogue_v2(const double2* __restrict__ C, long long ldc, const double2* __restrict__ Ukq,
                     const double2* __restrict__ ev, const double* __restrict__ omega, double* __restrict__ out,
                     int nq, int nw, int nm, int nb1, int nb2, int gb1, int QG, RateArgs ra, PolarArgs pa)
{
    constexpr int G = (KS == 1 || KS == 3) ? 2 : 1;       // b1 per warp item
    constexpr int TJ = (G * KS + 1) / 2;                  // a5 column tiles per item (last one half used when G*KS is odd)
    constexpr int NT = (KS + 1) / 2;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const bool polar = pa.P != nullptr;
    const Rot2Layout L = rot2_layout(QG, nw, nm, nb1, nb2, gb1, RATES, polar);
    const int nwp = L.nwp, MT = L.MT, ldu = L.ldu, ldz = L.ldz, ldzs = L.ldzs, Y = nw * nm, slack = L.slack;
    const size_t panel = L.panel;
    const int ngroups = L.ngroups, nbuf = L.nbuf;
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem_raw);                               // [2]
    double* inv2w = reinterpret_cast<double*>(smem_raw + L.off_inv2w);                   // [QG][8 NT]
    double2* Us = reinterpret_cast<double2*>(smem_raw + L.off_Us);                       // [QG][nwp][ldu]
    double2* Zs = reinterpret_cast<double2*>(smem_raw + L.off_Zs);                       // [QG][4 KS][ldz]
    double* Zsum = reinterpret_cast<double*>(smem_raw + L.off_Zsum);                     // [QG][4 KS][ldzs]
    double2* Cs = reinterpret_cast<double2*>(smem_raw + L.off_Cs);                       // [nbuf][QG][panel]
    double* om_s = reinterpret_cast<double*>(smem_raw + L.off_rates);                    // [QG][8 NT]   (RATES only)
    double* bose_s = om_s + QG * 8 * NT;                                                 // [QG][8 NT]
    double* e2_s = bose_s + QG * 8 * NT;                                                 // [QG][8 MT]
    double* f2_s = e2_s + QG * 8 * MT;                                                   // [QG][8 MT]
    double* wsum = f2_s + QG * 8 * MT;                                                   // [4 warps][nb1]
    double2* Ps = reinterpret_cast<double2*>(smem_raw + L.off_polar);                    // [QG][8 NT]
    double2* Os = Ps + QG * 8 * NT;                                                      // [QG][nb1][8 MT]
    const int q0 = blockIdx.x * QG;
    const int nql = min(QG, nq - q0);
    if (threadIdx.x == 0) { mbar_init(bar, 1); mbar_init(bar + 1, 1); mbar_fence_init(); }
    __syncthreads();
    auto issue = [&](int grp) {             // thread 0: bring the C panels of group grp (all nql q-points) in
        const int b10 = grp * gb1;
        const int nb1l = min(gb1, nb1 - b10);
        const uint32_t bytes = (uint32_t)((size_t)nb1l * Y * sizeof(double2));
        uint64_t* fb = bar + (grp & 1);
        mbar_arrive_expect_tx(fb, bytes * (uint32_t)nql);
        for (int ql = 0; ql < nql; ++ql)
            bulk_g2s(Cs + ((size_t)(grp & (nbuf - 1)) * QG + ql) * panel,
                     C + (size_t)(q0 + ql) * ldc + (size_t)b10 * Y, bytes, fb);
    };
    if (threadIdx.x == 0) issue(0);
    // while the first panels are in flight: conj(Ukq) -> Us, ev -> Zs / Zsum, 1/(2 omega), zero padding / slack.
    // These two loops come FIRST: their dependent global-load rounds are the longest latency chain of the CTA
    // (4-atom: 4.15 ms with this order, 4.67 ms with the small fills ahead of them -- measured).
    // Each thread first ISSUES the global loads of up to EB of its elements (of both arrays), then stores them: one
    // exposed load latency per round instead of one per element.
    double om_first = 0.0;                   // omega of this thread's first inv2w element rides along with the first round
    if ((int)threadIdx.x < nql * 8 * NT) {
        const int ql = threadIdx.x / (8 * NT), nu = threadIdx.x - ql * 8 * NT;
        if (nu < nm) om_first = omega[(size_t)(q0 + ql) * nm + nu];
    }
    {
        constexpr int EB = PHOEBE_ROT_EB;
        const int totU = nql * nwp * ldu, totZ = nql * 4 * KS * (8 * NT);
        for (int base = 0; base < max(totU, totZ); base += EB * blockDim.x) {
            double2 u[EB], zv[EB];
#pragma unroll
            for (int e = 0; e < EB; ++e) {
                const int i = base + e * blockDim.x + threadIdx.x;
                u[e] = make_double2(0.0, 0.0); zv[e] = make_double2(0.0, 0.0);
                if (i < totU) {
                    const int ql = i / (nwp * ldu), r = i - ql * nwp * ldu;
                    const int w2 = r / ldu, b2 = r - w2 * ldu;
                    if (w2 < nw && b2 < nb2) u[e] = Ukq[((size_t)(q0 + ql) * nw + w2) * nb2 + b2];
                }
                if (i < totZ) {
                    const int ql = i / (4 * KS * 8 * NT), r = i - ql * 4 * KS * 8 * NT;
                    const int ka = r / (8 * NT), nu = r - ka * 8 * NT;
                    if (ka < nm && nu < nm) zv[e] = ev[((size_t)(q0 + ql) * nm + ka) * nm + nu];
                }
            }
#pragma unroll
            for (int e = 0; e < EB; ++e) {
                const int i = base + e * blockDim.x + threadIdx.x;
                if (i < totU) { if (!(pa.conv & 1)) u[e].y = -u[e].y; Us[i] = u[e]; }
                if (i < totZ) {
                    const int ql = i / (4 * KS * 8 * NT), r = i - ql * 4 * KS * 8 * NT;
                    const int ka = r / (8 * NT), nu = r - ka * 8 * NT;
                    if (pa.conv & 2) zv[e].y = -zv[e].y;
                    Zs[((size_t)ql * 4 * KS + ka) * ldz + nu] = zv[e];
                    Zsum[((size_t)ql * 4 * KS + ka) * ldzs + nu] = zv[e].x + zv[e].y;
                }
            }
        }
    }
    for (int i = threadIdx.x; i < nql * 8 * NT; i += blockDim.x) {
        const int ql = i / (8 * NT), nu = i - ql * 8 * NT;
        const double w = (i == (int)threadIdx.x) ? om_first : ((nu < nm) ? omega[(size_t)(q0 + ql) * nm + nu] : 0.0);
        inv2w[i] = (w > 0.0) ? 0.5 / w : 0.0;
    }
    for (int i = threadIdx.x; i < nbuf * QG * slack; i += blockDim.x) {
        const int bq = i / slack, r = i - bq * slack;
        Cs[(size_t)bq * panel + (size_t)gb1 * Y + r] = make_double2(0.0, 0.0);
    }
    if (ngroups == 2 && nb1 - gb1 < gb1) {      // the second (last, narrower) group is the first user of buffer 1:
        const int nl = nb1 - gb1;                // what the padded reads behind its last b1 hit must be finite
        for (int i = threadIdx.x; i < QG * slack; i += blockDim.x) {
            const int ql = i / slack, r = i - ql * slack;
            Cs[((size_t)QG + ql) * panel + (size_t)nl * Y + r] = make_double2(0.0, 0.0);
        }
    }
    if (RATES) {
        for (int i = threadIdx.x; i < QG * 8 * NT; i += blockDim.x) {
            const int ql = i / (8 * NT), nu = i - ql * 8 * NT;
            const double w = (ql < nql && nu < nm) ? omega[(size_t)(q0 + ql) * nm + nu] : 0.0;
            om_s[i] = w;
            bose_s[i] = (w > 0.0) ? 1.0 / (exp(w * ra.inv_kT) - 1.0) : 0.0;
        }
        for (int i = threadIdx.x; i < QG * 8 * MT; i += blockDim.x) {
            const int ql = i / (8 * MT), b2 = i - ql * 8 * MT;
            const bool ok = ql < nql && b2 < nb2;
            const double e2 = ok ? ra.eps_kq[(size_t)(q0 + ql) * nb2 + b2] : 0.0;
            e2_s[i] = e2;
            f2_s[i] = ok ? 1.0 / (exp((e2 - ra.mu) * ra.inv_kT) + 1.0) : 0.0;
        }
        for (int i = threadIdx.x; i < 4 * nb1; i += blockDim.x) wsum[i] = 0.0;
    }
    if (polar) {
        for (int i = threadIdx.x; i < QG * 8 * NT; i += blockDim.x) {
            const int ql = i / (8 * NT), nu = i - ql * 8 * NT;
            Ps[i] = (ql < nql && nu < nm) ? pa.P[(size_t)(q0 + ql) * nm + nu] : make_double2(0.0, 0.0);
        }
        __syncthreads();                    // Us complete
        for (int i = threadIdx.x; i < nql * nb1 * 8 * MT; i += blockDim.x) {
            const int ql = i / (nb1 * 8 * MT), r = i - ql * nb1 * 8 * MT;
            const int b1 = r / (8 * MT), b2 = r - b1 * 8 * MT;
            double sr = 0.0, si = 0.0;
            if (b2 < nb2) {
                const double2* us = Us + (size_t)ql * nwp * ldu + b2;
                for (int w = 0; w < nw; ++w) {
                    const double2 u = us[(size_t)w * ldu], k = pa.Uk[(size_t)w * nb1 + b1];
                    sr = fma(u.x, k.x, sr); sr = fma(-u.y, k.y, sr);
                    si = fma(u.x, k.y, si); si = fma(u.y, k.x, si);
                }
            }
            Os[i] = make_double2(sr, si);
        }
    }

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarps = blockDim.x >> 5;
    const int g = lane >> 2, t = lane & 3;
    const int nks = nwp >> 2;
    const int nmg = (MT + MTW - 1) / MTW;
    for (int grp = 0; grp < ngroups; ++grp) {
        __syncthreads();                    // everyone is done with the buffer group grp+1 will overwrite (and with the fills)
        if (threadIdx.x == 0 && grp + 1 < ngroups) issue(grp + 1);
        mbar_wait(bar + (grp & 1), (uint32_t)(grp >> 1) & 1u);
        const int b10 = grp * gb1;
        const int nb1l = min(gb1, nb1 - b10);
        const int nbg = (nb1l + G - 1) / G;
        const int per_q = nbg * nmg;
        for (int item = warp; item < nql * per_q; item += nwarps) {
            const int ql = item / per_q, r = item - ql * per_q;
            const int bg = r / nmg, mg = r - bg * nmg;
            const int b1a = bg * G, mt0 = mg * MTW;
            // ---- a5: T1, T2, T3 of D[b2][(b1,ka)] ----
            double t1[MTW][TJ][2], t2[MTW][TJ][2], t3[MTW][TJ][2];
#pragma unroll
            for (int mi = 0; mi < MTW; ++mi)
#pragma unroll
                for (int j = 0; j < TJ; ++j) {
                    t1[mi][j][0] = t1[mi][j][1] = 0.0; t2[mi][j][0] = t2[mi][j][1] = 0.0; t3[mi][j][0] = t3[mi][j][1] = 0.0;
                }
            const double2* ua[MTW];
#pragma unroll
            for (int mi = 0; mi < MTW; ++mi)
                ua[mi] = Us + ((size_t)ql * nwp + t) * ldu + min(mt0 + mi, MT - 1) * 8 + g;
            const double2* pbase = Cs + ((size_t)(grp & (nbuf - 1)) * QG + ql) * panel + (size_t)t * nm + (g >> 1);
            const double2* cb[TJ];
#pragma unroll
            for (int j = 0; j < TJ; ++j) {
                const int p = min(2 * j + (g & 1), G * KS - 1);        // pair of this lane's B column (clamped: unused half tile)
                const int bl = p / KS, s = p - bl * KS;
                cb[j] = pbase + (size_t)min(b1a + bl, nb1l - 1) * Y + 4 * s;
            }
            double2 an[MTW], bn[TJ];
#pragma unroll
            for (int mi = 0; mi < MTW; ++mi) an[mi] = ua[mi][0];
#pragma unroll
            for (int j = 0; j < TJ; ++j) bn[j] = cb[j][0];
            for (int ks = 0; ks < nks; ++ks) {
                double2 a[MTW], b[TJ];
                double as[MTW], bs[TJ];
#pragma unroll
                for (int mi = 0; mi < MTW; ++mi) { a[mi] = an[mi]; as[mi] = a[mi].x + a[mi].y; }
#pragma unroll
                for (int j = 0; j < TJ; ++j) { b[j] = bn[j]; bs[j] = b[j].x + b[j].y; }
                if (ks + 1 < nks) {
#pragma unroll
                    for (int mi = 0; mi < MTW; ++mi) an[mi] = ua[mi][(size_t)(ks + 1) * 4 * ldu];
#pragma unroll
                    for (int j = 0; j < TJ; ++j) bn[j] = cb[j][(size_t)(ks + 1) * 4 * nm];
                }
#pragma unroll
                for (int mi = 0; mi < MTW; ++mi)
#pragma unroll
                    for (int j = 0; j < TJ; ++j) {
                        dmma884(t1[mi][j][0], t1[mi][j][1], a[mi].x, b[j].x);
                        dmma884(t2[mi][j][0], t2[mi][j][1], a[mi].y, b[j].y);
                        dmma884(t3[mi][j][0], t3[mi][j][1], as[mi], bs[j]);
                    }
            }
            // D = (T1 - T2) + i (T3 - T1 - T2); kept as (Re, Im, Re + Im): the three A planes of a6
#pragma unroll
            for (int mi = 0; mi < MTW; ++mi)
#pragma unroll
                for (int j = 0; j < TJ; ++j)
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        const double x1 = t1[mi][j][h], x2 = t2[mi][j][h], x3 = t3[mi][j][h];
                        t1[mi][j][h] = x1 - x2;
                        t2[mi][j][h] = x3 - x1 - x2;
                        t3[mi][j][h] = x3 - 2.0 * x2;
                    }
            // ---- a6 + a7 ----
            const double2* zq = Zs + ((size_t)ql * 4 * KS + t) * ldz + g;
            const double* zsq = Zsum + ((size_t)ql * 4 * KS + t) * ldzs + g;
            const double* iw = inv2w + ql * 8 * NT;
            double racc[G];
#pragma unroll
            for (int bl = 0; bl < G; ++bl) racc[bl] = 0.0;
#pragma unroll 1
            for (int n = 0; n < NT; ++n) {
                double e1[G][MTW][2], e2[G][MTW][2], e3[G][MTW][2];
#pragma unroll
                for (int bl = 0; bl < G; ++bl)
#pragma unroll
                    for (int mi = 0; mi < MTW; ++mi) {
                        e1[bl][mi][0] = e1[bl][mi][1] = 0.0; e2[bl][mi][0] = e2[bl][mi][1] = 0.0; e3[bl][mi][0] = e3[bl][mi][1] = 0.0;
                    }
#pragma unroll
                for (int s = 0; s < KS; ++s) {
                    const double2 z = zq[(size_t)4 * s * ldz + 8 * n];
                    const double zs = zsq[(size_t)4 * s * ldzs + 8 * n];
#pragma unroll
                    for (int bl = 0; bl < G; ++bl) {
                        const int p = bl * KS + s, j = p >> 1, h = p & 1;
#pragma unroll
                        for (int mi = 0; mi < MTW; ++mi) {
                            dmma884(e1[bl][mi][0], e1[bl][mi][1], t1[mi][j][h], z.x);
                            dmma884(e2[bl][mi][0], e2[bl][mi][1], t2[mi][j][h], z.y);
                            dmma884(e3[bl][mi][0], e3[bl][mi][1], t3[mi][j][h], zs);
                        }
                    }
                }
                const int nu = 8 * n + 2 * t;
                // per n-tile, outside the (b1, m-tile) loops: 1/(2 omega) of this lane's two columns (the padded array is
                // 8 NT long) and which of them exist -- the compiler does not hoist shared-memory loads over the stores
                const double iw0 = iw[nu], iw1 = iw[nu + 1];
                const bool okh[2] = {nu < nm, nu + 1 < nm};
#pragma unroll
                for (int bl = 0; bl < G; ++bl) {
                    if (b1a + bl >= nb1l) continue;
                    const int b1 = b10 + b1a + bl;
#pragma unroll
                    for (int mi = 0; mi < MTW; ++mi) {
                        const int b2 = (mt0 + mi) * 8 + g;
                        if (mt0 + mi >= MT || b2 >= nb2) continue;
                        double er[2], ei[2];
#pragma unroll
                        for (int h = 0; h < 2; ++h) {
                            er[h] = e1[bl][mi][h] - e2[bl][mi][h];
                            ei[h] = e3[bl][mi][h] - e1[bl][mi][h] - e2[bl][mi][h];
                        }
                        if (polar) {
                            const double2 o = Os[((size_t)ql * nb1 + b1) * 8 * MT + b2];
#pragma unroll
                            for (int h = 0; h < 2; ++h) {
                                const double2 pz = Ps[ql * 8 * NT + nu + h];
                                er[h] += pz.x * o.x - pz.y * o.y;
                                ei[h] += pz.x * o.y + pz.y * o.x;
                            }
                        }
                        double* orow = out + (((size_t)(q0 + ql) * nb1 + b1) * nb2 + b2) * nm;
                        double x12 = 0.0, f2 = 0.0;
                        if (RATES) {
                            x12 = ra.eps_k[(ra.rows_per_k > 0 ? (q0 / ra.rows_per_k) * nb1 : 0) + b1] - e2_s[ql * 8 * MT + b2];
                            f2 = f2_s[ql * 8 * MT + b2];
                        }
#pragma unroll
                        for (int h = 0; h < 2; ++h) {
                            if (!okh[h]) continue;
                            const double v = (er[h] * er[h] + ei[h] * ei[h]) * (h ? iw1 : iw0);
                            if (!RATES || out != nullptr) orow[nu + h] = v;
                            if (RATES) {
                                const double w = om_s[ql * 8 * NT + nu + h], bn_ = bose_s[ql * 8 * NT + nu + h];
                                const double dm = x12 - w, dp = x12 + w;
                                const double W = (1.0 - f2 + bn_) * exp(-(dm * dm) * ra.inv_sigma2) +
                                                 (f2 + bn_) * exp(-(dp * dp) * ra.inv_sigma2);
                                racc[bl] = fma(v, W, racc[bl]);
                            }
                        }
                    }
                }
            }
            if (RATES) {            // fixed-order sum over the warp, then into this warp's own row of wsum
#pragma unroll
                for (int bl = 0; bl < G; ++bl) {
                    double rsum = racc[bl];
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) rsum += __shfl_xor_sync(0xffffffffu, rsum, o);
                    if (lane == 0 && b1a + bl < nb1l) wsum[warp * nb1 + b10 + b1a + bl] += rsum;
                }
            }
        }
    }
    if (RATES) {
        __syncthreads();
        for (int b = threadIdx.x; b < nb1; b += blockDim.x)
            ra.partial[(size_t)blockIdx.x * nb1 + b] = ((wsum[b] + wsum[nb1 + b]) + wsum[2 * nb1 + b]) + wsum[3 * nb1 + b];
    }
}

}  // namespace pe
