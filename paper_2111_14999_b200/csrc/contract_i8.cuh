// contract_i8.cuh -- step a4 (Eq. 70) on the 5th-generation tensor cores (tcgen05.mma kind::i8, accumulators
// in TMEM) by exact integer splitting (the Ozaki scheme): B200's FP64 tensor pipe gives 37 TFLOP/s, its INT8 one 4.4 POP/s.
//
// The pair form (contract_pair.cuh) makes a4 a REAL GEMM  C'[q][n'] = sum_r A[q][r] B'[r][n'],  n' = (n, re|im).
// Every operand value is written as a 48-bit fixed-point number relative to a power-of-two scale (A: one scale for the
// whole phase matrix, |A| <= max weight; B': one scale per complex column n = twice the column's largest magnitude) and
// split into SIX balanced base-256 digits d_i in [-128, 127]:   x = scale * sum_i d_i 256^i / 2^47.
// Then  A B' = sA sB 2^-94 sum_{i,j} 256^(i+j) (A_i B'_j)  with A_i B'_j an INT8 x INT8 GEMM whose INT32 accumulation is
// EXACT (|sum| <= 6 pairs * rows * 128^2 < 2^31 for up to 16384 rows).  The 21 digit pairs with i + j >= 5 are kept, summed
// per level l = i + j - 5 in six TMEM accumulators; the dropped pairs are below 5 * 2^-48 of scale_A * scale_B per term -- a
// NORMWISE error, measured 3-5e-13 of max |g|^2 in the parity tests, inside the 1e-10 parity bar with two orders of magnitude
// to spare.  The levels
// are recombined exactly in 64-bit integers (two halves) and rounded once, in the FP64 epilogue that writes C in the
// layout the rotation kernel reads.
//
// Operands are produced ALREADY TILED for the tensor core (no-swizzle K-major canonical layout: core matrices of
// 8 rows x 16 bytes, 128 contiguous bytes each) with the six digit planes of a (tile, k chunk) side by side, so that a
// ring stage is TWO contiguous 1-D bulk copies (the TMA unit takes ~100 clk per bulk request whatever its size):
//   A digits  Ai8[m tile of 128][k chunk KC][d][row group 16][k group KC/16][8 rows][16 bytes]      (k_qphase_i8)
//   B digits  Bi8[slot][n' tile of 64][k chunk KC][d][col group 8][k group KC/16][8 cols][16 bytes]  (k_pack_i8)
// Kernel: warps 0..15 = epilogue (TMEM -> registers -> C), warp 16 = TMA producer, warp 17 = MMA issuer (one thread).
#pragma once
#include <math_constants.h>

#include "ptx_helpers.cuh"

namespace pe {

struct I8Cfg {
#ifndef PHOEBE_I8_KC
#define PHOEBE_I8_KC 32
#endif
    static constexpr int BM = 128, BN = 64, KC = PHOEBE_I8_KC, ND = 6, NLEV = 6, STAGES = 216 * 1024 / (ND * (BM + BN) * KC);
    static constexpr int EPI_WARPS = 16;
    // warps 0..15 = epilogue (four warpgroups), warps 16..19 = the control warpgroup: 16 = TMA producer, 17 = MMA issuer,
    // 18, 19 idle.  The register file is re-split at kernel start (setmaxnreg; pool = 640 threads x 96 at launch):
    // 512 x 112 + 128 x 32 = 61440.
    static constexpr int kThreads = (EPI_WARPS + 4) * 32, PW = EPI_WARPS, REGS_EPI = 112, REGS_CTRL = 32;
    static constexpr int A_PLANE = BM * KC, B_PLANE = BN * KC;                    // bytes of one digit plane of a stage
    static constexpr int STAGE_BYTES = ND * (A_PLANE + B_PLANE);                 // 36 KB (KC = 32): six stages
    static constexpr size_t kSmemBytes = (size_t)STAGES * STAGE_BYTES + 1024 + 256;   // + alignment slack + barriers
    static constexpr int TMEM_COLS = 512;                                        // NLEV * BN = 384 used
};

// six balanced base-256 digits of X = round(v * inv_scale * 2^47), |v * inv_scale| <= 1/2, as the six low BYTES of the result
// (byte i = digit i, a signed 8-bit number): with K = 128 (1 + 256 + ... + 256^5), Y = X + K is positive and below 2^48, its
// unsigned bytes y_i give X = sum_i (y_i - 128) 256^i, and y_i - 128 as int8 is y_i ^ 0x80 -- one add and one xor instead of
// six extract / subtract / shift rounds.
__device__ __forceinline__ unsigned long long i8_digits_packed(double v, double inv_scale)
{
    const long long X = __double2ll_rn(v * inv_scale * 140737488355328.0);       // 2^47
    return ((unsigned long long)X + 0x0000808080808080ULL) ^ 0x0000808080808080ULL;
}
// byte i (0..3) of each of four words -> one word (a's byte lowest)
template <int I>
__device__ __forceinline__ uint32_t i8_pick4(uint32_t a, uint32_t b, uint32_t c, uint32_t d)
{
    constexpr uint32_t sel = (uint32_t)I | ((uint32_t)(4 + I) << 4);
    return __byte_perm(__byte_perm(a, b, sel), __byte_perm(c, d, sel), 0x5410);
}
// digit plane I (0..5) of sixteen packed digit sets z[0..15] -> the 16 bytes of a core-matrix row
template <int I>
__device__ __forceinline__ int4 i8_plane16(const unsigned long long (&z)[16])
{
    uint32_t w[4];
#pragma unroll
    for (int g = 0; g < 4; ++g) {
        if (I < 4)
            w[g] = i8_pick4<(I & 3)>((uint32_t)z[4 * g], (uint32_t)z[4 * g + 1], (uint32_t)z[4 * g + 2], (uint32_t)z[4 * g + 3]);
        else
            w[g] = i8_pick4<(I & 3)>((uint32_t)(z[4 * g] >> 32), (uint32_t)(z[4 * g + 1] >> 32), (uint32_t)(z[4 * g + 2] >> 32),
                                     (uint32_t)(z[4 * g + 3] >> 32));
    }
    return make_int4((int)w[0], (int)w[1], (int)w[2], (int)w[3]);
}

// byte offset of element (row, k) of digit 0 in the tiling [row tile][k chunk][digit][row group][k group][8][16];
// digit d is d * rows_per_tile * KC bytes further
__device__ __forceinline__ size_t i8_tiled_off(int row, int k, int rows_per_tile, int nchunks)
{
    constexpr int KC = I8Cfg::KC;
    const int tile = row / rows_per_tile, rl = row - tile * rows_per_tile;
    const int chunk = k / KC, kl = k - chunk * KC;
    return ((size_t)tile * nchunks + chunk) * (size_t)(I8Cfg::ND * rows_per_tile * KC) +
           (size_t)(((rl >> 3) * (KC / 16) + (kl >> 4)) * 128 + (rl & 7) * 16 + (kl & 15));
}

// A digits.  Row order of the pair form (k_qphase_pair): cosine rows r < Kc (pairs first), sine row of pair sl at Kc16 + sl
// (Kc16 = the cosine block padded to a multiple of 16, so a thread's 16 cosine rows and their 16 sine rows are whole
// 16-byte groups).  One thread = one q-point x 16 consecutive cosine rows.  Columns q >= nq are zero digits; the 16-row groups
// behind the sine block are never written (the planes are zeroed once at setup).
// grid (ceil(ldq/128), ceil(Kc16/16)), block 128.
__global__ void __launch_bounds__(128)
k_qphase_i8(const double* __restrict__ q, const double* __restrict__ Rrow, const double* __restrict__ wrow, int K2, int Kc,
            int Kc16, int nq, int Kpad, int ldq, double sgn, double inv_scaleA, int8_t* __restrict__ Ai8)
{
    const int iq = blockIdx.x * 128 + threadIdx.x;
    if (iq >= ldq) return;
    const int r0 = blockIdx.y * 16;
    const int nchunks = Kpad / I8Cfg::KC;
    double q0 = 0.0, q1 = 0.0, q2 = 0.0;
    const bool valid = iq < nq;
    if (valid) { q0 = q[3 * (size_t)iq]; q1 = q[3 * (size_t)iq + 1]; q2 = q[3 * (size_t)iq + 2]; }
    unsigned long long zc[16], zs[16];
#pragma unroll
    for (int u = 0; u < 16; ++u) {
        const int r = r0 + u;
        double vc = 0.0, vs = 0.0;
        if (valid && r < Kc) {
            const double x = q0 * Rrow[3 * r] + q1 * Rrow[3 * r + 1] + q2 * Rrow[3 * r + 2];
            double sn, cs;
            sincospi(2.0 * x, &sn, &cs);
            vc = wrow[r] * cs; vs = (r < K2) ? wrow[r] * sgn * sn : 0.0;
        }
        zc[u] = i8_digits_packed(vc, inv_scaleA);
        zs[u] = i8_digits_packed(vs, inv_scaleA);
    }
    const size_t oc = i8_tiled_off(iq, r0, I8Cfg::BM, nchunks);
    const bool has_sin = r0 < K2;                          // the sine group of these 16 rows exists
    const size_t os = has_sin ? i8_tiled_off(iq, Kc16 + r0, I8Cfg::BM, nchunks) : 0;
#define PE_I8_STORE_PLANE(I)                                                                                     \
    *reinterpret_cast<int4*>(Ai8 + (size_t)(I) * I8Cfg::A_PLANE + oc) = i8_plane16<I>(zc);                       \
    if (has_sin) *reinterpret_cast<int4*>(Ai8 + (size_t)(I) * I8Cfg::A_PLANE + os) = i8_plane16<I>(zs);
    PE_I8_STORE_PLANE(0) PE_I8_STORE_PLANE(1) PE_I8_STORE_PLANE(2) PE_I8_STORE_PLANE(3) PE_I8_STORE_PLANE(4) PE_I8_STORE_PLANE(5)
#undef PE_I8_STORE_PLANE
}

// column maxima of B': cmax[slot][n] = max_r |pair row r of column n| (re or im), as the bit pattern of the non-negative
// double (ordered like the integers) under atomicMax; zeroed by the host before the launch.  One thread = one column x 16
// rows.  grid (ceil(N/128), ceil(Kr/16), nslots), block 128.
__global__ void __launch_bounds__(128)
k_i8_colmax(const double2* __restrict__ g1, long long ld, long long strideS, int N, int Kr, const int* __restrict__ pa,
            const int* __restrict__ pb, const int* __restrict__ kind, unsigned long long* __restrict__ cmax, int ldsb)
{
    const int n = blockIdx.x * 128 + threadIdx.x, slot = blockIdx.z, r0 = blockIdx.y * 16;
    if (n >= N) return;
    const double2* s = g1 + (size_t)slot * strideS + n;
    double m = 0.0;
#pragma unroll 4
    for (int r = r0; r < min(r0 + 16, Kr); ++r) {
        if (kind[r] == 2) continue;
        const double2 a = s[(size_t)pa[r] * ld];
        const int ib = pb[r];
        const double2 b = ib >= 0 ? s[(size_t)ib * ld] : make_double2(0.0, 0.0);
        const double x = kind[r] == 0 ? a.x + b.x : a.y - b.y, y = kind[r] == 0 ? a.y + b.y : a.x - b.x;
        m = fmax(m, fmax(fabs(x), fabs(y)));
        if (!(isfinite(x) && isfinite(y))) m = CUDART_INF;        // NaN / Inf in g1': the whole column becomes NaN (as in FP64)
    }
    if (m > 0.0) atomicMax(cmax + (size_t)slot * ldsb + n, (unsigned long long)__double_as_longlong(m));
}

// column scale from the maximum: 2^(e+1) with 2^e > m (m = f 2^e, f in [1/2, 1)); 1 for an all-zero column
__device__ __forceinline__ double i8_scale_of(unsigned long long mbits)
{
    const double m = __longlong_as_double((long long)mbits);
    if (!(m > 0.0)) return 1.0;
    if (isinf(m)) return m;          // a non-finite column: digits 0 (1 / inf), result 0 * inf = NaN
    int e = 0;
    frexp(m, &e);
    return ldexp(1.0, e + 1);
}

// B' digits: real column n' = 2 n + c (c = 0: re, 1: im) of pair row r, relative to the column scale sb[slot][n] (written here
// from the column maximum).  One thread = one real column x 16 consecutive rows.
// grid (ceil(Npad2/128), Kpad/16, nslots), block 128.  Columns >= 2 N and rows >= Kr are zero digits.
__global__ void __launch_bounds__(128)
k_pack_i8(const double2* __restrict__ g1, long long ld, long long strideS, int N, int Npad2, int Kr, int Kpad,
          const int* __restrict__ pa, const int* __restrict__ pb, const int* __restrict__ kind,
          const unsigned long long* __restrict__ cmax, double* __restrict__ sb, int ldsb, int8_t* __restrict__ Bi8,
          size_t slot_bytes)
{
    const int np = blockIdx.x * 128 + threadIdx.x, slot = blockIdx.z;
    if (np >= Npad2) return;
    const int n = np >> 1, c = np & 1, r0 = blockIdx.y * 16;
    const bool colok = n < N;
    const double scale = colok ? i8_scale_of(cmax[(size_t)slot * ldsb + n]) : 1.0;
    const double inv = colok ? 1.0 / scale : 0.0;
    if (colok && c == 0 && blockIdx.y == 0) sb[(size_t)slot * ldsb + n] = scale;      // the GEMM epilogue's column scale
    const double2* s = g1 + (size_t)slot * strideS + (colok ? n : 0);
    unsigned long long z[16];
#pragma unroll
    for (int u = 0; u < 16; ++u) {
        const int r = r0 + u;
        double v = 0.0;
        if (colok && r < Kr && kind[r] != 2) {
            const double2 a = s[(size_t)pa[r] * ld];
            const int ib = pb[r];
            const double2 b = ib >= 0 ? s[(size_t)ib * ld] : make_double2(0.0, 0.0);
            if (kind[r] == 0) v = c ? a.y + b.y : a.x + b.x;            // a + b
            else v = c ? a.x - b.x : -(a.y - b.y);                      // i (a - b)
        }
        z[u] = i8_digits_packed(v, inv);
    }
    int8_t* dst = Bi8 + (size_t)slot * slot_bytes + i8_tiled_off(np, r0, I8Cfg::BN, Kpad / I8Cfg::KC);
    *reinterpret_cast<int4*>(dst + 0 * (size_t)I8Cfg::B_PLANE) = i8_plane16<0>(z);
    *reinterpret_cast<int4*>(dst + 1 * (size_t)I8Cfg::B_PLANE) = i8_plane16<1>(z);
    *reinterpret_cast<int4*>(dst + 2 * (size_t)I8Cfg::B_PLANE) = i8_plane16<2>(z);
    *reinterpret_cast<int4*>(dst + 3 * (size_t)I8Cfg::B_PLANE) = i8_plane16<3>(z);
    *reinterpret_cast<int4*>(dst + 4 * (size_t)I8Cfg::B_PLANE) = i8_plane16<4>(z);
    *reinterpret_cast<int4*>(dst + 5 * (size_t)I8Cfg::B_PLANE) = i8_plane16<5>(z);
}

// ---- tcgen05 helpers (PTX ISA: tcgen05.*, sm_100a) -------------------------------------------------------------------
// shared-memory matrix descriptor, K-major, no swizzle: core matrices of 8 rows x 16 bytes; lbo = byte distance between
// core matrices adjacent in K, sbo = between those adjacent in M / N (verified against a host product on this B200)
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo)
{
    return (uint64_t)((saddr >> 4) & 0x3FFF) | ((uint64_t)((lbo >> 4) & 0x3FFF) << 16) | ((uint64_t)((sbo >> 4) & 0x3FFF) << 32) |
           ((uint64_t)1 << 46);
}
__device__ __forceinline__ void umma_i8(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, {%5, %5, %5, %5}, p;\n\t}\n"
                 :: "r"(tmem_d), "l"(da), "l"(db), "r"(idesc), "r"(accumulate), "r"(0u) : "memory");
}
// The same, executed by ALL lanes of the (converged) MMA warp with the instruction itself predicated on `leader`: inside an
// `if (lane == 0)` branch ptxas cannot prove the descriptors warp-uniform and wraps every tcgen05.mma in an ELECT / R2UR
// broadcast loop (~20 instructions per MMA).  Predicated in converged code, with the stage address made uniform by a shuffle,
// the descriptors are computed in uniform registers.  (Measured: the kernel time did not change -- the issuing thread was
// not the limit, it blocks on the tensor pipe's queue -- the lighter instruction stream is kept.)
__device__ __forceinline__ void umma_i8_p(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate, uint32_t leader)
{
    asm volatile("{\n\t.reg .pred p, q;\n\tsetp.ne.b32 p, %4, 0;\n\tsetp.ne.b32 q, %6, 0;\n\t"
                 "@q tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, {%5, %5, %5, %5}, p;\n\t}\n"
                 :: "r"(tmem_d), "l"(da), "l"(db), "r"(idesc), "r"(accumulate), "r"(0u), "r"(leader) : "memory");
}
__device__ __forceinline__ void umma_commit_p(uint64_t* bar, uint32_t leader)
{
    asm volatile("{\n\t.reg .pred q;\n\tsetp.ne.b32 q, %1, 0;\n\t"
                 "@q tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n\t}\n"
                 :: "r"(smem_u32(bar)), "r"(leader) : "memory");
}
__device__ __forceinline__ void umma_commit_mc_p(uint64_t* bar, uint16_t cta_mask, uint32_t leader)
{
    asm volatile("{\n\t.reg .pred q;\n\tsetp.ne.b32 q, %2, 0;\n\t"
                 "@q tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;\n\t}\n"
                 :: "r"(smem_u32(bar)), "h"(cta_mask), "r"(leader) : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t* bar)      // arrives on bar when all MMAs issued so far have completed
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void umma_commit_mc(uint64_t* bar, uint16_t cta_mask)   // ... on bar of every CTA in cta_mask
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
                 :: "r"(smem_u32(bar)), "h"(cta_mask) : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&r)[16])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
                   "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                 : "r"(taddr));
}

// 16 TMEM lanes x 16 columns in the matrix-fragment shape: lane t gets rows t/4 and t/4 + 8, column pairs 2 (t%4) + {0, 1} and
// 8 + 2 (t%4) + {0, 1}: r[0..1] = (row t/4, pair t%4), r[2..3] = (row t/4 + 8, same pair), r[4..7] the same for the pair 4 + t%4
// (layout read back from the hardware with a tcgen05.st / tcgen05.ld probe)
__device__ __forceinline__ void tmem_ld_16x256b_x2(uint32_t taddr, uint32_t (&r)[8])
{
    asm volatile("tcgen05.ld.sync.aligned.16x256b.x2.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                 : "r"(taddr));
}

// C[q][n] (complex, layout CMap) = sum_r A[q][r] B'[r][(n, re|im)] from the digit planes.  M rows of A (q), N complex
// columns, Kpad (multiple of 64) rows; Ai8 / Bi8 tiled as above (plane strides in bytes); sb = column scales of this slot.
// rowsPerB > 0: stacked multi-k form, rows [j rowsPerB, (j+1) rowsPerB) use B slot j (rowsPerB a multiple of 128).
// CL > 1: launched in clusters of CL CTAs that work on CL neighbouring column tiles of the SAME row tile: each CTA fetches
// 1/CL of the A digit planes of a stage and multicasts it to the whole cluster (the A planes are 2/3 of a stage: L2 -> SM
// traffic per tile 884 KB -> 590 KB (CL = 2), 442 KB (CL = 4)); a stage is refilled when every CTA of the cluster has
// released it (tcgen05.commit multicast onto every CTA's empty barrier).
template <int CL>
__global__ void __launch_bounds__(I8Cfg::kThreads, 1)
k_contract_i8(const int8_t* __restrict__ Ai8, const int8_t* __restrict__ Bi8, size_t b_slot_bytes, const double* __restrict__ sb, int ldsb, double scaleA, double2* __restrict__ C,
              long long ldc, int M, int N, int Kpad, int rowsPerB, int rowOffset, CMap cm)
{
    using Cfg = I8Cfg;
    constexpr int BM = Cfg::BM, BN = Cfg::BN, KC = Cfg::KC, ND = Cfg::ND, ST = Cfg::STAGES;
    extern __shared__ unsigned char smem_dyn[];
    unsigned char* smem = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_dyn) + 1023) & ~(uintptr_t)1023);
    uint64_t* full = reinterpret_cast<uint64_t*>(smem + (size_t)ST * Cfg::STAGE_BYTES);
    uint64_t* empty = full + ST;
    uint64_t* tfull = empty + ST;           // accumulators of a tile complete
    uint64_t* tempty = tfull + 1;           // accumulators read out by the epilogue
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tempty + 1);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < ST; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, CL); }
        mbar_init(tfull, 1); mbar_init(tempty, Cfg::EPI_WARPS);
        mbar_fence_init();
    }
    if (warp == Cfg::PW + 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" :: "r"(smem_u32(tmem_slot)), "r"(Cfg::TMEM_COLS));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (CL > 1) cluster_sync_all();                     // the peers' barriers exist before anything is multicast to them
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = *tmem_slot;
    const int nchunks = Kpad / KC;
    const int ntn = (2 * N + BN - 1) / BN, ntm = (M + BM - 1) / BM;
    // tile groups of CL neighbouring column tiles, n fastest: the CTAs running together share a few A row blocks
    const int ntng = (ntn + CL - 1) / CL;
    const int ngroups = ntng * ntm;
    // Order of the tile groups: PANELS of as many column groups as there are CTAs (clusters) in flight, all row tiles of a
    // panel before the next panel -- a CTA keeps its column tile while the row tiles go by, so the B digits of a panel
    // (148 x 64 columns x Kpad x 6 B <= 44 MB) stay in L2 however wide g1' is (large: 141 MB of B digits per slot were
    // re-read from DRAM for every row tile in the plain n-fastest order: 11.7 GB per launch), and the A tile of the moment
    // is shared by all CTAs.
    const int pw = min(CL > 1 ? (int)cluster_nid_x() : (int)gridDim.x, ntng);
    auto group_tile = [&](int g, int& tm, int& tng) {
        const int per_panel = pw * ntm, panel = g / per_panel, r = g - panel * per_panel;
        const int w = min(pw, ntng - panel * pw);          // the last panel may be narrower
        tm = r / w;
        tng = panel * pw + (r - tm * w);
    };
    const int crank = CL > 1 ? (int)cluster_ctarank() : 0;
    const int g0 = CL > 1 ? (int)cluster_id_x() : (int)blockIdx.x, gstep = CL > 1 ? (int)cluster_nid_x() : (int)gridDim.x;
    constexpr uint16_t kMask = (uint16_t)((1u << CL) - 1u);
    constexpr int A_STAGE = ND * Cfg::A_PLANE, B_STAGE = ND * Cfg::B_PLANE;

    if (warp >= Cfg::PW) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(Cfg::REGS_CTRL));
    if (warp == Cfg::PW) {
        // ================= TMA producer: two contiguous bulk copies per stage =================
        int s = 0; uint32_t ph = 0;
        for (int g = g0; g < ngroups; g += gstep) {
            int tm, tng;
            group_tile(g, tm, tng);
            const int tn = min(tng * CL + crank, ntn - 1);                          // a tile past the edge re-reads the last one
            const int slot = rowsPerB > 0 ? (rowOffset + tm * BM) / rowsPerB : 0;
            const int8_t* a_src = Ai8 + (size_t)tm * nchunks * A_STAGE;
            const int8_t* b_src = Bi8 + (size_t)slot * b_slot_bytes + (size_t)tn * nchunks * B_STAGE;
            for (int c = 0; c < nchunks; ++c) {
                mbar_wait(empty + s, ph ^ 1u);
                unsigned char* st = smem + (size_t)s * Cfg::STAGE_BYTES;
                if (lane == 0) {
                    mbar_arrive_expect_tx(full + s, (uint32_t)Cfg::STAGE_BYTES);
                    if (CL == 1) bulk_g2s(st, a_src + (size_t)c * A_STAGE, A_STAGE, full + s);
                    else         // this CTA's 1/CL of the A planes, to every CTA of the cluster
                        bulk_g2s_mc(st + crank * (A_STAGE / CL), a_src + (size_t)c * A_STAGE + crank * (A_STAGE / CL), A_STAGE / CL,
                                    full + s, kMask);
                    bulk_g2s(st + A_STAGE, b_src + (size_t)c * B_STAGE, B_STAGE, full + s);
                }
                __syncwarp();
                if (++s == ST) { s = 0; ph ^= 1u; }
            }
        }
    } else if (warp == Cfg::PW + 1) {
        // ================= MMA issuer (one elected lane; the warp stays converged) =================
        // Digit plane A_i meets the B' planes j = 5 - i .. 5, whose products belong to the levels 0 .. i: the planes are
        // contiguous in the stage and the level accumulators contiguous in TMEM, so ONE instruction with N = 64 (i + 1)
        // does all of them and reads the A tile from shared memory once (the unit's limit is N <= 256: i = 4 and 5 take two).
        // Shared-memory reads per 32-deep step: 75 KB instead of the 126 KB of 21 single-level instructions.  With the 36 KB
        // the TMA unit writes per step that is 111 KB = 867 clk at the SM's 128 B/clk, against 725 clk of tensor-pipe time:
        // the kernel is bound by shared-memory bandwidth (measured: 925-966 clk per step, tensor pipe 68 % active).
        // instruction descriptor: D = S32, A = B = signed 8 bit, both K-major, M = 128, N in bits 17..22
        constexpr uint32_t idesc0 = (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(BM >> 4) << 24);
        int s = 0; uint32_t ph = 0, tph = 0;
        const uint32_t tmem_u = __shfl_sync(0xffffffffu, tmem, 0);
        for (int g = g0; g < ngroups; g += gstep) {
            mbar_wait(tempty, tph ^ 1u);                 // the epilogue has read the previous tile's accumulators
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            for (int c = 0; c < nchunks; ++c) {
                mbar_wait(full + s, ph);
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                {
                    const uint32_t leader = lane == 0 ? 1u : 0u;
                    // (a shuffle from lane 0 tells the compiler the address is warp-uniform: the descriptor arithmetic then runs
                    //  in uniform registers)
                    const uint32_t a0 = __shfl_sync(0xffffffffu, smem_u32(smem + (size_t)s * Cfg::STAGE_BYTES), 0), b0 = a0 + ND * Cfg::A_PLANE;
#pragma unroll
                    for (int ks = 0; ks < KC / 32; ++ks) {
                        const uint32_t acc = (c == 0 && ks == 0) ? 0u : 1u;
                        // i = 5 first: its two instructions initialise all six levels of a new tile
#pragma unroll
                        for (int i = ND - 1; i >= 0; --i) {
                            const uint64_t da = umma_desc(a0 + i * Cfg::A_PLANE + ks * 256, 128, (KC / 16) * 128);
                            const int j0 = ND - 1 - i, nlev = i + 1;              // planes j0 .. 5 -> levels 0 .. i
                            // more than four levels exceed N = 256: split 3 + rest (N = 192 + 128 / 192 runs faster than 256 + 64 / 128:
                            // a narrow instruction is bound by its shared-memory reads of the A tile)
                            const int n1 = nlev > 4 ? 3 : nlev;
                            umma_i8_p(tmem_u, da, umma_desc(b0 + j0 * Cfg::B_PLANE + ks * 256, 128, (KC / 16) * 128),
                                      idesc0 | ((uint32_t)((n1 * BN) >> 3) << 17), i == ND - 1 ? acc : 1u, leader);
                            if (nlev > 4)
                                umma_i8_p(tmem_u + 3u * BN, da, umma_desc(b0 + (j0 + 3) * Cfg::B_PLANE + ks * 256, 128, (KC / 16) * 128),
                                          idesc0 | ((uint32_t)(((nlev - 3) * BN) >> 3) << 17), i == ND - 1 ? acc : 1u, leader);
                        }
                    }
                    // frees the stage (in every CTA of the cluster) when these MMAs have read it
                    if (CL == 1) umma_commit_p(empty + s, leader); else umma_commit_mc_p(empty + s, kMask, leader);
                    if (c == nchunks - 1) umma_commit_p(tfull, leader);
                }
                __syncwarp();
                if (++s == ST) { s = 0; ph ^= 1u; }
            }
            tph ^= 1u;
        }
    }
    } else {
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(Cfg::REGS_EPI));
        // ================= epilogue warps (16): TMEM lanes 32 (warp % 4) .. + 31 = rows; column group cg = 16 real columns ===
        // Each warp pulls the six levels of its 32 x 16 block into registers (96 raw INT32 per thread, tcgen05.ld in the
        // 16x256b fragment shape) and hands the
        // accumulators back to the MMA warp AT ONCE: only the TMEM read-out itself is not overlapped with the next tile's
        // MMAs (six levels x 64 columns = 384 of the 512 TMEM columns leave no room for a second accumulator set).  The exact
        // recombination in 64-bit integers, the scaling and the stores then run beside the MMAs.  Column offsets (CMap) and
        // scales are computed once per tile by lanes 0..7 and broadcast.
        constexpr int CW = BN / (Cfg::EPI_WARPS / 4);               // real columns per warp: 16
        static_assert(CW == 16, "two tcgen05.ld 16x256b.x2 per level and warp");
        const int wq = warp & 3, cg = warp >> 2;
        uint32_t tph = 0;
        const double kscale = scaleA * 5.551115123125783e-17;        // 2^-54
        for (int g = g0; g < ngroups; g += gstep) {
            int tm, tng;
            group_tile(g, tm, tng);
            const int tn = tng * CL + crank;                                        // tn >= ntn: nothing to store
            const int slot = rowsPerB > 0 ? (rowOffset + tm * BM) / rowsPerB : 0;
            const int ncol = tn * (BN / 2) + cg * (CW / 2) + (lane & 7);    // this lane's complex column (lanes 8..31 mirror)
            long long off_l = -1; double sc_l = 0.0;
            if (ncol < N) { off_l = cmap_off(ncol, cm); sc_l = kscale * sb[(size_t)slot * ldsb + ncol]; }
            uint32_t v[Cfg::NLEV][2][8];                  // [level][16-lane half][fragment register]
            mbar_wait(tfull, tph);
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
            for (int l = 0; l < Cfg::NLEV; ++l)
#pragma unroll
                for (int hh = 0; hh < 2; ++hh)
                    tmem_ld_16x256b_x2(tmem + ((uint32_t)(wq * 32 + 16 * hh) << 16) + (uint32_t)(l * BN + cg * CW), v[l][hh]);
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            __syncwarp();
            if (lane == 0) mbar_arrive(tempty);
            tph ^= 1u;
            // In the fragment shape four neighbouring lanes hold four neighbouring complex columns of ONE row: a store
            // instruction writes 8 rows x 64 contiguous bytes (whole 32-byte sectors) instead of 32 rows x 16 bytes.
#pragma unroll
            for (int cs = 0; cs < 2; ++cs) {
                const int csrc = cs * 4 + (lane & 3);                   // this lane's complex column of the warp's eight
                const long long off = __shfl_sync(0xffffffffu, off_l, csrc);
                const double sc = __shfl_sync(0xffffffffu, sc_l, csrc);
#pragma unroll
                for (int hh = 0; hh < 2; ++hh) {
#pragma unroll
                    for (int rs = 0; rs < 2; ++rs) {
                        const int m = tm * BM + wq * 32 + 16 * hh + 8 * rs + (lane >> 2);
                        double val[2];
#pragma unroll
                        for (int h = 0; h < 2; ++h) {
                            const int e = cs * 4 + rs * 2 + h;
                            const long long lo = (long long)(int)v[0][hh][e] + ((long long)(int)v[1][hh][e] << 8) + ((long long)(int)v[2][hh][e] << 16);
                            const long long hi = (long long)(int)v[3][hh][e] + ((long long)(int)v[4][hh][e] << 8) + ((long long)(int)v[5][hh][e] << 16);
                            // int64 -> double on the integer pipe plus one DADD (instead of I2F.F64.S64): for |x| < 2^51
                            // the bit pattern of 1.5 * 2^52 plus x IS the double 1.5 * 2^52 + x; with the exponent raised by 24, + 2^24 x
                            const double lod = __longlong_as_double(lo + 0x4338000000000000LL) - 6755399441055744.0;
                            const double hid = __longlong_as_double(hi + 0x4338000000000000LL + (24LL << 52)) - 6755399441055744.0 * 16777216.0;
                            val[h] = hid + lod;                        // = hi 2^24 + lo, exact up to this one rounding
                        }
                        if (m < M && off >= 0) C[(size_t)m * ldc + off] = make_double2(val[0] * sc, val[1] * sc);
                    }
                }
            }
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (CL > 1) cluster_sync_all();                     // no CTA leaves while a peer may still multicast into it
    if (warp == Cfg::PW + 1) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem), "r"(Cfg::TMEM_COLS));
}

}  // namespace pe
