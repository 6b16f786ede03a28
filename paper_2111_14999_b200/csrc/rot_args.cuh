// rot_args.cuh -- argument structs shared by the rotation kernels (rotate_v3.cuh and the plain fallback in
// qbatch_kernels.cuh) and their translation units.
#pragma once
#include <cuda_runtime.h>

namespace pe {

// ---------------------------------------------------------------------------
// Arguments shared by the rotation kernels (rotate_v3.cuh; the plain fallback below).
//
// RATES (Eq. 29 L229 with the Gaussian delta of Eq. 61): every |g|^2 value is also
// multiplied by the occupation/energy-conservation bracket
//   W = (1 - f' + n) G(eps_k[b1] - omega - eps_kq[q][b2]) + (f' + n) G(eps_k[b1] + omega - eps_kq[q][b2]),
//   G(x) = exp(-x^2/sigma^2),  f' = 1/(e^{(eps_kq - mu)/kT} + 1),  n = 1/(e^{omega/kT} - 1)
// and summed over (b2, nu) in a fixed order into partial rows; k_rate_reduce adds the partial rows (fixed order) times
// pref/(sqrt(pi) sigma) into rate[b1].  `out` may then be nullptr (|g|^2 is not stored).
// ---------------------------------------------------------------------------
struct RateArgs {
    const double* eps_k;    // [nb1]; stacked form: [k slots][nb1], the slot of a q-point = (its row) / rows_per_k
    const double* eps_kq;   // [nq][nb2] (of this launch)
    double inv_kT, mu, inv_sigma2;
    double* partial;        // rotate_v3: [nq][nmg][nb1], one row per (q, group of b2 tiles); plain path: [chunks][nb1]
    int rows_per_k;         // > 0: the q lists of several k slots are stacked
};

// f4 (Eq. 14-15): when pa.P != nullptr the long-range amplitude P[q][nu] * O[q][b1][b2],
// O = sum_w conj(Ukq[q][w][b2]) Uk[w][b1] (the overlap [U_kq^dagger U_k]_{b2 b1}), is added to E before |.|^2.
// rotate_v3 forms O on the tensor cores as one more column tile of a5 (B = U_k instead of the C panel).
struct PolarArgs {
    const double2* P;     // [nq][nm] of this launch, or nullptr
    const double2* Uk;    // [nw][nb1]
    int conv;             // set_conventions: bit 0 = U_kq enters PLAIN (default: conjugated), bit 1 = ev enters CONJUGATED
};

}  // namespace pe
