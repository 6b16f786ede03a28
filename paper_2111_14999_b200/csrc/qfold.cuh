// qfold.cuh -- the q <-> -q fold of step a4 (Eq. 70 on uniform meshes, L282 / L669: fine q meshes are closed under
// inversion).  In the pair form (contract_pair.cuh) the phase rows are real: cosine rows are EVEN in q, sine rows ODD, so
//     C(q) = Ce(q) + Co(q),   C(-q) = Ce(q) - Co(q),     Ce = sum over cosine rows, Co = sum over sine rows
// and one pass over the rows of a representative q gives both q and -q: half the contraction for a list closed under
// inversion.  -q is meant modulo a reciprocal lattice vector when every Rp is an integer vector (the phases are then
// periodic, Eq. 87), else literally.
//
// k_qfold_detect (ONE CTA; its hash table lives in shared memory for lists of up to 8192 q-points) finds the pairs on the
// device, with no host round trip: a hash table of the canonical coordinates, a lookup of every q-point's negative,
// mutual-partner marking, and an index-ordered compaction of the representatives.  meta[0] = number of representatives, meta[1] = 1 if the fold pays (>= 25 % fewer rows), else 0: the
// kernels of both paths are launched and the ones whose path is not taken return at once.  Everything is deterministic
// (duplicates resolve to the smallest index).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace pe {

__device__ __forceinline__ unsigned long long qfold_bits(double x, int integer_rp, double sgn)
{
    double v = sgn * x;
    if (integer_rp) v = v - floor(v);            // canonical fractional part in [0, 1)
    v += 0.0;                                    // -0 -> +0
    return (unsigned long long)__double_as_longlong(v);
}
__device__ __forceinline__ unsigned int qfold_hash(unsigned long long a, unsigned long long b, unsigned long long c)
{
    unsigned long long h = a * 0x9E3779B97F4A7C15ull;
    h ^= (b + 0x9E3779B97F4A7C15ull + (h << 6) + (h >> 2));
    h *= 0xC2B2AE3D27D4EB4Full;
    h ^= (c + 0x165667B19E3779F9ull + (h << 6) + (h >> 2));
    h ^= h >> 29; h *= 0xBF58476D1CE4E5B9ull; h ^= h >> 32;
    return (unsigned int)h;
}

// One CTA.  Work arrays: table [tsize] (a power of two >= 2 nq), partner [nq], fp [nq] (64-bit fingerprints of the
// canonical coordinates) -- in shared memory when they fit (in_smem: nq <= 8192), else the global scratch passed in.
// Outputs (global): rep_idx [nq], mate [nq], meta [2].
__global__ void __launch_bounds__(1024)
k_qfold_detect(const double* __restrict__ q, int nq, int integer_rp, int in_smem, int* __restrict__ g_table, int tsize,
               int* __restrict__ g_partner, unsigned long long* __restrict__ g_fp, int* __restrict__ rep_idx,
               int* __restrict__ mate, int* __restrict__ meta)
{
    extern __shared__ __align__(16) unsigned char qf_smem[];
    __shared__ int s_warp[32];
    const int tid = threadIdx.x, nt = blockDim.x, lane = tid & 31, wid = tid >> 5;
    unsigned long long* fp = in_smem ? reinterpret_cast<unsigned long long*>(qf_smem) : g_fp;
    int* table = in_smem ? reinterpret_cast<int*>(qf_smem + (size_t)nq * 8) : g_table;
    int* partner = in_smem ? table + tsize : g_partner;
    const unsigned int mask = (unsigned int)tsize - 1u;
    for (int i = tid; i < tsize; i += nt) table[i] = -1;
    auto bits3 = [&](int j, double sg, unsigned long long& a, unsigned long long& b, unsigned long long& c) {
        a = qfold_bits(q[3 * (size_t)j], integer_rp, sg); b = qfold_bits(q[3 * (size_t)j + 1], integer_rp, sg);
        c = qfold_bits(q[3 * (size_t)j + 2], integer_rp, sg);
    };
    // (mesh points have only a few high mantissa bits set: every component goes through a full 64-bit finaliser)
    auto fmix = [](unsigned long long x) {
        x ^= x >> 33; x *= 0xff51afd7ed558ccdull; x ^= x >> 33; x *= 0xc4ceb9fe1a85ec53ull; x ^= x >> 33;
        return x;
    };
    auto fingerprint = [&](unsigned long long a, unsigned long long b, unsigned long long c) {
        return fmix(fmix(fmix(a + 0x9E3779B97F4A7C15ull) ^ b) ^ c);
    };
    for (int i = tid; i < nq; i += nt) {
        unsigned long long a, b, c;
        bits3(i, 1.0, a, b, c);
        fp[i] = fingerprint(a, b, c);
    }
    __syncthreads();
    // insert: a slot ends up holding the SMALLEST index among q-points with equal coordinates (fingerprints filter, the
    // coordinates decide)
    for (int i = tid; i < nq; i += nt) {
        const unsigned long long f = fp[i];
        unsigned int slot = (unsigned int)f & mask;
        for (;;) {
            const int old = atomicCAS(&table[slot], -1, i);
            if (old == -1) break;
            if (fp[old] == f) {
                unsigned long long a, b, c, a2, b2, c2;
                bits3(i, 1.0, a, b, c); bits3(old, 1.0, a2, b2, c2);
                if (a == a2 && b == b2 && c == c2) { atomicMin(&table[slot], i); break; }
            }
            slot = (slot + 1) & mask;
        }
    }
    __syncthreads();
    // lookup of -q
    for (int i = tid; i < nq; i += nt) {
        unsigned long long a, b, c;
        bits3(i, -1.0, a, b, c);
        const unsigned long long f = fingerprint(a, b, c);
        unsigned int slot = (unsigned int)f & mask;
        int found = -1;
        for (;;) {
            const int j = table[slot];
            if (j == -1) break;
            if (fp[j] == f) {
                unsigned long long a2, b2, c2;
                bits3(j, 1.0, a2, b2, c2);
                if (a == a2 && b == b2 && c == c2) { found = j; break; }
            }
            slot = (slot + 1) & mask;
        }
        partner[i] = found;
    }
    __syncthreads();
    // representatives in index order: i follows p(i) iff p(i) < i and the partnership is mutual.  Every thread owns a
    // contiguous range of q-points: count, block-wide exclusive scan of the counts, scatter.
    const int per = (nq + nt - 1) / nt;
    const int i0 = min(nq, tid * per), i1 = min(nq, i0 + per);
    int cnt = 0;
    for (int i = i0; i < i1; ++i) {
        const int p = partner[i];
        cnt += !(p >= 0 && p != i && p < i && partner[p] == i);
    }
    int incl = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
    }
    if (lane == 31) s_warp[wid] = incl;
    __syncthreads();
    if (wid == 0) {
        int w = lane < (nt >> 5) ? s_warp[lane] : 0, wi = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, wi, o);
            if (lane >= o) wi += v;
        }
        s_warp[lane] = wi - w;                       // exclusive prefix of the warp totals
        if (lane == 31) { meta[0] = wi; meta[1] = (4LL * wi <= 3LL * nq) ? 1 : 0; }
    }
    __syncthreads();
    int pos = s_warp[wid] + incl - cnt;
    for (int i = i0; i < i1; ++i) {
        const int p = partner[i];
        const bool mutual = p >= 0 && p != i && partner[p] == i;
        if (!(mutual && p < i)) { rep_idx[pos] = i; mate[pos] = (mutual && p > i) ? p : -1; ++pos; }
    }
}

}  // namespace pe
