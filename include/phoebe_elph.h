/*
 * phoebe_elph.h -- C ABI of the B200-native el-ph Wannier->Bloch |g|^2 hot path.
 *
 * What the library computes (PAPER.md = /root/reference/PAPER.md, the Phoebe
 * paper, arXiv 2111.14999):
 *
 *   Eq. 13 (L133)  g0(k,q) = sum_{Re,Rp} e^{ik.Re + iq.Rp} U_{k+q} g0(Re,Rp) U_k^dagger z_q
 *   Eq. 7  (L98)   g = (1 / (2 m omega_{q nu}))^{1/2} g0
 *   Eq. 70-71 (L564-L570)  the factorisation: a fixed-k precompute, then the
 *                  completion for a set {k'} batched on the GPU (L576)
 *
 * in the reading fixed by SURVEY.md 8(c) / DESIGN.md "Readings":
 *
 *   out[q][b1][b2][nu] = | sum_{e,p} (e^{2 pi i k.Re_e}/deg_e[e]) (e^{2 pi i q.Rp_p}/deg_p[p])
 *                           sum_{w1,w2,kappa} U_k[w1][b1] conj(U_kq[q][w2][b2]) ev[q][kappa][nu]
 *                           g_W[p][e][w1][w2][kappa] |^2  /  (2 omega[q][nu])        (0 where omega <= 0)
 *
 * Conventions
 *   - every array is C-order (last index fastest); complex128 = (re, im) pair
 *     of doubles, 16-byte aligned; wavevectors and lattice vectors are in
 *     crystal (fractional) coordinates (L510), hence the explicit 2 pi.
 *   - "DEVICE" pointers are CUDA device pointers on the current device,
 *     "HOST" pointers are ordinary host memory.  BORROWED = the caller keeps
 *     ownership and must keep the memory valid until the stream given at
 *     setup has finished the work of the call that used it.
 *   - every call only enqueues work on that stream and returns (no implicit
 *     device synchronisation) unless its comment says otherwise.
 *   - return value: 0 = OK, negative = error (see PHOEBE_ELPH_E_*).  The
 *     library never aborts, throws or prints.  There is no CPU fallback: on a
 *     machine without a CUDA device every compute call fails with
 *     PHOEBE_ELPH_E_CUDA.
 */
#ifndef PHOEBE_ELPH_H
#define PHOEBE_ELPH_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PHOEBE_ELPH_OK            0
#define PHOEBE_ELPH_E_NULL       -1   /* a required pointer is NULL                        */
#define PHOEBE_ELPH_E_DIMS       -2   /* a dimension is <= 0 or exceeds its declared max   */
#define PHOEBE_ELPH_E_ALIGN      -3   /* a complex / workspace pointer is not 16-B aligned */
#define PHOEBE_ELPH_E_NO_K       -4   /* q_batch called before any set_k                   */
#define PHOEBE_ELPH_E_WORKSPACE  -5   /* workspace too small for these dims                */
#define PHOEBE_ELPH_E_CUDA       -6   /* CUDA error; text via phoebe_elph_last_error       */

typedef struct phoebe_elph_ctx phoebe_elph_ctx;     /* opaque, library-owned */

/* Problem sizes (paper's notation):
 * nRe/nRp electron/phonon lattice vectors, nw Wannier functions, nmodes = 3*atoms,
 * nb1_max/nb2_max = most bands ever kept at k / at k+q (<= nw), nq_max = most
 * q-points ever passed to one q_batch call. */
typedef struct {
    int32_t nRe, nRp, nw, nmodes, nb1_max, nb2_max, nq_max;
    int32_t nk_max;   /* most k-points per phoebe_elph_set_k_batch (0 or 1 = single-k only; <= 32) */
} phoebe_elph_dims;

/* Kernel kinds, for launch counts and profiling. */
enum {
    PHOEBE_ELPH_K_SETK_STREAM = 0,  /* a1: Fourier sum over Re (streams g_W once)         */
    PHOEBE_ELPH_K_SETK_ROTATE = 1,  /* a2: rotation by U_k -> g1'                          */
    PHOEBE_ELPH_K_QPHASE      = 2,  /* a3: phases e^{2 pi i q.Rp}/deg_p                    */
    PHOEBE_ELPH_K_CONTRACT    = 3,  /* a4: Rp contraction (complex FP64 GEMM, DMMA)        */
    PHOEBE_ELPH_K_ROTATE_EPI  = 4,  /* a5-a7: U_kq^dagger, phonon rotation, |.|^2/(2 omega) */
    PHOEBE_ELPH_K_SETK_GEMM   = 5,  /* a1 for a batch of k: one pass over g_W (FP64 GEMM, DMMA) */
    PHOEBE_ELPH_K_RATE_REDUCE = 6,  /* f2: fixed-order sum of the per-CTA linewidth partials    */
    PHOEBE_ELPH_K_POLAR       = 7,  /* f4: (q, nu) amplitudes of the polar long-range term        */
    PHOEBE_ELPH_K_PACK        = 8,  /* g1' -> planar blocked operand of the planar contraction    */
    PHOEBE_ELPH_K_QFOLD       = 9,  /* a4 on inversion-symmetric q lists: detection of the (q, -q) pairs  */
    PHOEBE_ELPH_K_COUNT       = 10
};

/* Size the workspace (L576: "the size of the set {k'} is optimized at runtime so
 * that most of the on-board GPU's memory is used").
 * In : dims (dims->nq_max may be 0 = "as many as fit"), hbm_budget_bytes = device
 *      bytes the caller can give to the workspace (g_W itself excluded).
 * Out: *nq_batch_out = largest q-batch that fits (<= dims->nq_max when that is > 0),
 *      *bytes_out    = workspace bytes needed for that batch size.
 * Errors: E_NULL, E_DIMS, E_WORKSPACE (budget too small for even one tile of q). */
int phoebe_elph_workspace_bytes(const phoebe_elph_dims* dims, size_t hbm_budget_bytes,
                                size_t* bytes_out, int32_t* nq_batch_out);

/* Step a0.  Creates a context bound to one device stream.
 *   gW_dev      DEVICE, BORROWED for the life of ctx, complex128 [nRp][nRe][nw][nw][nmodes]
 *               (first Wannier index <-> k / U_k, second <-> k+q / U_kq; Eq. 13).
 *               Never copied or re-laid-out (57.8 GB in the largest workload).
 *   Re_host     HOST [nRe][3], Rp_host HOST [nRp][3]: lattice vectors, crystal coords; copied.
 *   deg_e_host  HOST [nRe], deg_p_host HOST [nRp]: Wigner-Seitz degeneracies (> 0), each
 *               Fourier term is divided by them; NULL = all 1; copied.
 *   dims->nq_max must be > 0 here.
 *   workspace_dev DEVICE, BORROWED for the life of ctx, >= phoebe_elph_workspace_bytes(), 256-B aligned.
 *   cuda_stream a cudaStream_t (NULL = default stream).
 * Synchronises the stream once (the small copies use pageable host memory).
 *   At setup the library also pairs every Rp vector with its inverse -R (exact match, equal degeneracy): step a4 then
 *   runs as real (cos | sin) phase rows times complex rows g1'[R] + g1'[-R], i (g1'[R] - g1'[-R]) -- see tuning "pair".
 *   Any list is accepted; vectors without partner cost two rows instead of one.  Re / Rp must be finite (E_DIMS).
 * Errors: E_NULL, E_DIMS, E_ALIGN, E_WORKSPACE, E_CUDA. */
int phoebe_elph_setup(phoebe_elph_ctx** ctx_out, const void* gW_dev,
                      const double* Re_host, const double* Rp_host,
                      const double* deg_e_host, const double* deg_p_host,
                      const phoebe_elph_dims* dims,
                      void* workspace_dev, size_t workspace_bytes, void* cuda_stream);

/* Steps a1 + a2, Eq. 71 (L570):
 *   g1'[p][b1][w2][kappa] = sum_{w1} U_k[w1][b1] sum_e (e^{2 pi i k.Re_e}/deg_e[e]) g_W[p][e][w1][w2][kappa]
 * kept inside the context for the following q_batch calls.
 *   k_host  HOST [3] (read before returning);  Uk_dev DEVICE complex128 [nw][nb1], columns = eigenvectors
 *   (Eq. 11), 1 <= nb1 <= nb1_max; nb1 may change from call to call (band windows, L540).
 * Errors: E_NULL, E_DIMS, E_ALIGN, E_CUDA. */
int phoebe_elph_set_k(phoebe_elph_ctx* ctx, const double* k_host, const void* Uk_dev, int32_t nb1);

/* Same, U_k in HOST memory (copied to the device on the stream; the host buffer
 * may be reused when the call returns only if it is pageable -- for pinned memory
 * keep it valid until the stream has passed the copy). */
int phoebe_elph_set_k_host(phoebe_elph_ctx* ctx, const double* k_host, const void* Uk_host, int32_t nb1);

/* Steps a1 + a2 for a BATCH of k-points in one pass over g_W.  Eq. 71 (L570) is
 * "precomputed at fixed k" once per k, which re-reads all of g_W (0.5 flop/byte) for every k; here the
 * Fourier sum over Re of nk k-points is one [nk x nRe].[nRe x nw*nw*nmodes] complex GEMM per phonon
 * vector, so g_W is read once per batch.  Results are identical to nk set_k calls up to rounding order.
 *   nk <= dims.nk_max;  k_host HOST [nk][3] (read before returning);
 *   Uk_dev DEVICE complex128 [nk][nw][nb1] (same nb1 for the whole batch).
 * The g1' of all nk k-points stay in the context; q_batch uses the one chosen by
 * phoebe_elph_select_k (index 0 right after this call).  A later set_k overwrites slot 0.
 * Errors: E_NULL, E_DIMS, E_ALIGN, E_CUDA. */
int phoebe_elph_set_k_batch(phoebe_elph_ctx* ctx, int32_t nk, const double* k_host, const void* Uk_dev, int32_t nb1);
int phoebe_elph_set_k_batch_host(phoebe_elph_ctx* ctx, int32_t nk, const double* k_host, const void* Uk_host, int32_t nb1);

/* Make the g1' of k-point i (0 <= i < nk of the last set_k_batch) the one q_batch uses.  Host-side only.
 * Errors: E_NULL, E_NO_K, E_DIMS. */
int phoebe_elph_select_k(phoebe_elph_ctx* ctx, int32_t i);

/* Steps a3..a7, rest of Eq. 70 + Eq. 7, for nq q-points at the k of the last set_k:
 *   C[q][b1][w2][kappa] = sum_p (e^{2 pi i q.Rp_p}/deg_p[p]) g1'[p][b1][w2][kappa]
 *   D[q][b1][b2][kappa] = sum_{w2} conj(U_kq[q][w2][b2]) C[q][b1][w2][kappa]
 *   E[q][b1][b2][nu]    = sum_kappa D[q][b1][b2][kappa] ev[q][kappa][nu]
 *   out[q][b1][b2][nu]  = |E|^2 / (2 omega[q][nu])      (0 where omega <= 0)
 *   q_dev DEVICE [nq][3]; Ukq_dev DEVICE complex128 [nq][nw][nb2]; ev_dev DEVICE complex128
 *   [nq][nmodes][nmodes] (row kappa = 3*atom+cartesian, column nu = mode; used unconjugated, any
 *   1/sqrt(mass) folded in by the caller); omega_dev DEVICE [nq][nmodes];
 *   out_dev DEVICE double [nq][nb1][nb2][nmodes], written, caller-owned.
 *   0 <= nq <= nq_max, 1 <= nb2 <= nb2_max (uniform within the batch).  nq = 0 (an empty batch) is a no-op in
 *   every q_batch* entry point: returns OK, no pointer is read, nothing is written, `rate` is left as it is.
 * Errors: E_NULL, E_DIMS, E_ALIGN, E_NO_K, E_CUDA. */
int phoebe_elph_q_batch(phoebe_elph_ctx* ctx, int32_t nq, int32_t nb2,
                        const double* q_dev, const void* Ukq_dev, const void* ev_dev,
                        const double* omega_dev, double* out_dev);

/* q_batch for the first nk k slots of the last set_k_batch in ONE pass (one phase, one contraction and one rotation
 * launch for all of them): the inputs / outputs of the k slots are stacked, k slowest --
 *   q_dev [nk][nq][3], Ukq_dev [nk][nq][nw][nb2], ev_dev [nk][nq][nmodes][nmodes], omega_dev [nk][nq][nmodes],
 *   out_dev [nk][nq][nb1][nb2][nmodes];  rows of slot j are contracted with the g1' of slot j.
 * Results are identical to nk select_k + q_batch calls.  It exists for band windows with few bands (L526-540), where
 * one k-point's q list is too small a GEMM to fill 148 SMs.  nq must be a multiple of 64, nk*nq <= dims.nq_max;
 * not available while the polar term is switched on.
 * Errors: E_NULL, E_NO_K, E_DIMS, E_ALIGN, E_CUDA. */
int phoebe_elph_q_batch_multi(phoebe_elph_ctx* ctx, int32_t nk, int32_t nq, int32_t nb2,
                              const double* q_dev, const void* Ukq_dev, const void* ev_dev,
                              const double* omega_dev, double* out_dev);

/* Same with HOST buffers: copies the four inputs host->device into staging inside the
 * workspace, runs the batch, copies out device->host, and SYNCHRONISES the stream before
 * returning (so pageable buffers are safe).  This is the end-to-end call. */
int phoebe_elph_q_batch_host(phoebe_elph_ctx* ctx, int32_t nq, int32_t nb2,
                             const double* q_host, const void* Ukq_host, const void* ev_host,
                             const double* omega_host, double* out_host);

/* Pipelined form of q_batch_host (the paper moves every batch of |g|^2 back to the CPU, L556 / L707; here the
 * copies overlap the kernels): enqueues the four host->device copies on a copy-in stream, the batch on the
 * compute stream and the device->host copy of out on a copy-out stream, chained by events, over two staging
 * slots inside the workspace, and RETURNS WITHOUT WAITING -- the copy-in of batch n+1 and the copy-out of
 * batch n-1 run while batch n computes.  The host buffers must be page-locked (cudaHostAlloc / pinned) for
 * the overlap and must stay valid and unmodified (inputs) / unread (out_host) until phoebe_elph_wait returns;
 * with pageable memory the copies are staged by the driver and the call degrades to q_batch_host's ordering.
 * set_k / set_k_batch / select_k may be called between batches (they are ordered on the compute stream).
 * Errors: as q_batch_host. */
int phoebe_elph_q_batch_host_async(phoebe_elph_ctx* ctx, int32_t nq, int32_t nb2,
                                   const double* q_host, const void* Ukq_host, const void* ev_host,
                                   const double* omega_host, double* out_host);

/* Blocks until every batch enqueued by q_batch_host_async has been copied out (and the compute stream is idle).
 * Errors: E_NULL, E_CUDA. */
int phoebe_elph_wait(phoebe_elph_ctx* ctx);

/* q_batch with the linewidth sum fused into the |g|^2 epilogue (no |g|^2 round trip
 * to the host; the paper does this sum on the CPU, L556 / L707).  Eq. 29 (L229) with the Gaussian delta
 * of Eq. 61 (L437), delta(k-k'+q) resolved by k' = k+q, hbar = 1:
 *   rate[b1] += pref * sum_{q<nq, b2<nb2, nu<nmodes} out[q][b1][b2][nu] *
 *               [ (1 - f(eps_kq[q][b2]) + n(omega[q][nu])) d(eps_k[b1] - omega[q][nu] - eps_kq[q][b2])
 *               + (    f(eps_kq[q][b2]) + n(omega[q][nu])) d(eps_k[b1] + omega[q][nu] - eps_kq[q][b2]) ]
 *   f(e) = 1/(exp((e - mu)/kT) + 1),  n(w) = 1/(exp(w/kT) - 1),  d(x) = exp(-x^2/sigma^2)/(sqrt(pi) sigma);
 *   terms with omega <= 0 contribute nothing.  `pref` carries the paper's 2 pi/(N_k V) and any unit factor.
 *   eps_k_dev DEVICE [nb1] band energies at k; eps_kq_dev DEVICE [nq][nb2] band energies at k+q;
 *   rate_dev DEVICE [nb1], ACCUMULATED INTO (the caller zeroes it before the first batch of a k-point);
 *   out_dev as in q_batch, or NULL: |g|^2 is then not stored at all.
 * The sum runs in a fixed order: results are bit-reproducible for a given batch split.
 * Errors: as q_batch, plus E_DIMS when kT <= 0 or sigma <= 0. */
typedef struct { double kT, mu, sigma, pref; } phoebe_elph_rate_params;
int phoebe_elph_q_batch_rates(phoebe_elph_ctx* ctx, int32_t nq, int32_t nb2,
                              const double* q_dev, const void* Ukq_dev, const void* ev_dev, const double* omega_dev,
                              const double* eps_k_dev, const double* eps_kq_dev, const phoebe_elph_rate_params* prm,
                              double* rate_dev, double* out_dev);

/* q_batch_rates for the first nk k slots of the last set_k_batch in ONE pass (the stacked form of q_batch_multi: one
 * phase, one contraction, one rotation + linewidth launch): the use the paper describes -- scattering rates of the bands
 * in a window around the chemical potential (L526-540, Eq. 29) for many k-points, where one k-point's q list is too small
 * a GEMM for 148 SMs.  Arrays stacked, k slowest: q_dev [nk][nq][3], Ukq_dev [nk][nq][nw][nb2], ev_dev [nk][nq][nmodes][nmodes],
 * omega_dev [nk][nq][nmodes], eps_k_dev [nk][nb1], eps_kq_dev [nk][nq][nb2], rate_dev [nk][nb1] (ACCUMULATED INTO),
 * out_dev [nk][nq][nb1][nb2][nmodes] or NULL.  Results equal nk select_k + q_batch_rates calls up to the rounding order of
 * the sum (fixed, reproducible).  nq a multiple of 64, nk*nq <= dims.nq_max and small enough for one contraction launch
 * (E_DIMS otherwise), nmodes <= 48, polar term off.
 * Errors: E_NULL, E_NO_K, E_DIMS, E_ALIGN, E_CUDA. */
int phoebe_elph_q_batch_rates_multi(phoebe_elph_ctx* ctx, int32_t nk, int32_t nq, int32_t nb2,
                                    const double* q_dev, const void* Ukq_dev, const void* ev_dev, const double* omega_dev,
                                    const double* eps_k_dev, const double* eps_kq_dev, const phoebe_elph_rate_params* prm,
                                    double* rate_dev, double* out_dev);

/* Pipelined HOST forms of the two stacked calls (a single small call is latency-bound, so batch; L707: the
 * results go back to the CPU): the k-stacked arrays of a whole set_k_batch in PINNED host memory, same layout as the device
 * forms.  Like q_batch_host_async they return at once: the copy-in of batch n+1 (its own stream) and the copy-out of batch
 * n-1 (its own stream) overlap the kernels of batch n -- and so does the next set_k_batch, which runs on the compute stream
 * behind this batch's kernels while its results are still being copied out.  Host arrays (and rate_host, out_host) must
 * stay valid and untouched until phoebe_elph_wait; at most two batches are in flight.
 * Errors: as the device forms. */
int phoebe_elph_q_batch_multi_host_async(phoebe_elph_ctx* ctx, int32_t nk, int32_t nq, int32_t nb2, const double* q_host,
                                         const void* Ukq_host, const void* ev_host, const double* omega_host,
                                         double* out_host);
int phoebe_elph_q_batch_rates_multi_host_async(phoebe_elph_ctx* ctx, int32_t nk, int32_t nq, int32_t nb2,
                                               const double* q_host, const void* Ukq_host, const void* ev_host,
                                               const double* omega_host, const double* eps_k_host,
                                               const double* eps_kq_host, const phoebe_elph_rate_params* prm,
                                               double* rate_host /* [nk][nb1], accumulated into */,
                                               double* out_host /* [nk][nq][nb1][nb2][nmodes] or NULL */);

/* Same with HOST buffers (rate_host [nb1] is read, accumulated into and written back; out_host may be
 * NULL, and then only nb1 doubles come back); SYNCHRONISES the stream before returning. */
int phoebe_elph_q_batch_rates_host(phoebe_elph_ctx* ctx, int32_t nq, int32_t nb2,
                                   const double* q_host, const void* Ukq_host, const void* ev_host,
                                   const double* omega_host, const double* eps_k_host, const double* eps_kq_host,
                                   const phoebe_elph_rate_params* prm, double* rate_host, double* out_host);

/* Pipelined form of q_batch_rates_host, on the same two staging slots and streams as q_batch_host_async (the two may
 * be mixed; phoebe_elph_wait ends both).  rate_host [nb1] is read when the call is made, accumulated into on the device
 * and written back by the copy-out stream: give every call in flight its OWN rate array (e.g. one per k-point) and read it
 * after phoebe_elph_wait.  out_host may be NULL.  Host buffers should be page-locked.
 * Errors: as q_batch_rates_host. */
int phoebe_elph_q_batch_rates_host_async(phoebe_elph_ctx* ctx, int32_t nq, int32_t nb2,
                                         const double* q_host, const void* Ukq_host, const void* ev_host,
                                         const double* omega_host, const double* eps_k_host, const double* eps_kq_host,
                                         const phoebe_elph_rate_params* prm, double* rate_host, double* out_host);

/* Copy the current g1' (complex128 [nRp][nb1][nw][nmodes]) to dst_dev (DEVICE, >= bytes
 * nRp*nb1*nw*nmodes*16); for tests of set_k on its own.  Errors: E_NULL, E_NO_K, E_WORKSPACE, E_CUDA. */
int phoebe_elph_copy_g1(phoebe_elph_ctx* ctx, void* dst_dev, size_t dst_bytes);

/* polar (long-range) correction, Eq. 14-15 (L139-L147): g = g^S + g^L.  After this call every
 * q_batch / q_batch_rates (and their host forms) adds, to the amplitude of Eq. 13 before |.|^2,
 *   L[q][b1][b2][nu] = P[q][nu] * sum_w conj(U_kq[q][w][b2]) U_k[w][b1]            (overlap [U_kq^dagger U_k])
 *   P[q][nu] = i coeff sum_{G in list, q+G != 0} (Q . Zeff_nu) / (Q . eps_inf . Q),   Q = (q + G) . recip,
 *   Zeff_nu[a] = sum_{s,b} Zstar[s][a][b] ev[q][3s+b][nu]
 * (readings R20-R24 of DESIGN.md: 1/sqrt(m_s) is inside ev, 1/sqrt(2 omega) is the final 1/(2 omega), everything
 * else of Eq. 15's prefactor is the real `coeff`; no convergence factor is applied -- the caller chooses the G list).
 *   recip_host HOST [3][3] rows = reciprocal lattice vectors (Cartesian); G_host HOST [nG][3] crystal coordinates,
 *   0 <= nG <= 4096, nG = 0 switches the term off (the other pointers may then be NULL);
 *   Zstar_host HOST [nmodes/3][3][3] Born effective charges; eps_inf_host HOST [3][3].  All copied; synchronises
 *   the stream once.  nmodes must be a multiple of 3.
 * Errors: E_NULL, E_DIMS, E_CUDA. */
int phoebe_elph_set_polar(phoebe_elph_ctx* ctx, const double* recip_host, int32_t nG, const double* G_host,
                          const double* Zstar_host, const double* eps_inf_host, double coeff);

/* the second workload with the Eq. 70 shape: the three-phonon coupling of Eq. 5 (L82; L137, L558:
 * "either three phonon and electron-phonon scattering ... a tensor operation in the form" of Eq. 70).  Eq. 70 is one
 * contraction; what differs between its two uses is the sign of the Fourier phases and which rotation matrices enter
 * conjugated.  Defaults = the el-ph reading of Eq. 13: phase_sign = +1, U_k plain, U_kq conjugated, ev plain.
 * Eq. 5 (readings R25-R27):  phase_sign = -1 and all three conjugated, with
 *   g_W := V3[R'][R][a][b][c] (complex128), Re := R, Rp := R', nw = nmodes = 3 x atoms,
 *   set_k(q, z_q [nm][n0]),  q_batch(q', z_{q'} [nq][nm][n1], z_{q''} [nq][nm][nm], omega := 0.5)  ->
 *   out[q'][nu][nu'][nu''] = |sum_{R,R'} e^{-2 pi i (q.R + q'.R')} sum_{abc} z*[a][nu] z'*[b][nu'] z''*[c][nu''] V3|^2
 * (mass / frequency factors of Eq. 5 folded into the eigenvectors by the caller, as in q_batch; with omega = 0.5 the
 * final 1/(2 omega) is 1).  Invalidates the current set_k.  Not combinable with the polar term.
 * Errors: E_NULL, E_DIMS. */
int phoebe_elph_set_conventions(phoebe_elph_ctx* ctx, int32_t phase_sign, int32_t conj_Uk, int32_t conj_Ukq,
                                int32_t conj_ev);

/* the paper's "pool" (L576): when g(Re,Rp) does not fit one GPU it is distributed over Re.
 * Eq. 71 is linear in g_W, so a rank that was set up with ITS Re vectors and ITS slab g_W[nRp][nRe_local][...]
 * gets from set_k / set_k_batch the partial g1' of its shard; the sum over the ranks is the g1' of Eq. 71.
 * This call hands out the g1' storage inside the workspace so that the caller can sum it IN PLACE across ranks
 * (ncclAllReduce / torch.distributed.all_reduce on the context's stream) before q_batch:
 *   slot >= 0: *ptr_out = DEVICE address of the g1' of k slot `slot` (complex128 [nRp][nb1][nw][nmodes]),
 *              *bytes_out = nRp*nb1*nw*nmodes*16;
 *   slot = -1: the storage of all k slots filled by the last set_k / set_k_batch as one range (slots are
 *              *stride_out bytes apart; the gap after each slot's data is padding and may be summed along).
 * stride_out may be NULL.  Host-side only.  Errors: E_NULL, E_NO_K, E_DIMS. */
int phoebe_elph_g1_buffer(phoebe_elph_ctx* ctx, int32_t slot, void** ptr_out, size_t* bytes_out, size_t* stride_out);

/* Launch accounting: counts[PHOEBE_ELPH_K_COUNT] = kernels launched so far, per kind. */
int phoebe_elph_launch_counts(const phoebe_elph_ctx* ctx, int64_t* counts);

/* Per-kernel device timing.  profile(ctx, 1) starts recording a CUDA event pair around
 * every kernel launch on the context's stream (a few microseconds of overhead per launch:
 * do not time whole-job throughput with it on); profile_read synchronises the stream,
 * returns accumulated milliseconds and launch counts per kind since the last read and
 * clears them.  profile(ctx, 0) stops recording. */
int phoebe_elph_profile(phoebe_elph_ctx* ctx, int32_t enable);
int phoebe_elph_profile_read(phoebe_elph_ctx* ctx, double* ms, int64_t* launches);

/* Tuning knobs (integers); unknown key -> E_DIMS.  Keys:
 *   "nq_sub"    q-points per contraction / rotation launch (default: the whole batch when C fits); rounded down to a
 *               multiple of 128 (at least 128), so that no contraction row tile straddles two sub-batches or k slots
 *   "s_split"   number of Re chunks in the set_k stream (0 = automatic)
 *   "m3"        1 (default) = three-multiply complex product in the two GEMMs (T1 = Ar.Br, T2 = Ai.Bi,
 *               T3 = (Ar+Ai).(Br+Bi); Re = T1-T2, Im = T3-T1-T2: 6 instead of 8 real flop per complex MAC,
 *               normwise FP64-accurate); 0 = the four-multiply product
 *   "tile"      contraction CTA tile: 0 = automatic (cost model), 32 or 64
 *   "planar"    1 (default) = a4 through the planar-operand contraction (re / im / re+im planes blocked by 64
 *               columns, one LDS.128 feeds two DMMA tiles, no operand-sum DADDs); 0 = the interleaved-complex kernel
 *   "pair"      1 (default) = a4 in the +R / -R pair form (real cos / sin phase rows x complex rows g1'[p] + g1'[pbar],
 *               i (g1'[p] - g1'[pbar]): 4 real flop per complex MAC, exact) whenever the Rp list has enough inversion
 *               pairs (4 Kr < 6 nRp, Kr = real rows: 2 per pair or partner-less vector, 1 for R = 0); 0 = never; 2 = whenever
 *               the rows fit the operand buffers (Kr <= 1.5 nRp).  get_tuning("pair_rows") = Kr if the last contraction
 *               launch used the form, else 0.   "pair_ctas" 1 | 2 = persistent CTAs per SM of that kernel
 *   "i8"        1 (default) = the pair form of a4 runs on the INT8 tensor cores (tcgen05.mma kind::i8, accumulators in
 *               TMEM) by EXACT digit splitting: each FP64 operand is rounded to 48 bits relative to a power-of-two scale
 *               (one for the phase matrix, one per column of g1') and written as six signed base-256 digits; the 21 digit
 *               pairs of weight >= 256^5 are INT8 GEMMs with exact INT32 accumulation, recombined in 64-bit integers and
 *               rounded once.  Normwise error ~1e-13 of a column's largest entry, results
 *               bit-reproducible.  Taken whenever the pair form is and (stacked forms) the rows per k-point are a multiple
 *               of 128; 0 = the FP64 tensor-core pair kernel.  get_tuning("i8") = 1 if the LAST contraction ran on INT8.
 *               Domain: column maxima of g1' within ~[1e-290, 1e290]; a NaN / Inf in g1' turns its whole column of the
 *               contraction (hence every |g|^2 that column enters) into NaN, as FP64 arithmetic would.  The q-points must be
 *               finite (a NaN wavevector gives undefined phase digits, not NaN).
 *               "i8_cluster" 0 | 1 (default) | 2 | 4 | 8 = CTAs per cluster of that kernel (the A digit planes multicast);
 *               get_tuning("i8_grid") = CTAs of the last launch (clusters of 8: 15 fit a B200 = 120 CTAs)
 *   "qfold"     1 = q lists that contain -q with q (uniform meshes; modulo a reciprocal lattice vector when all Rp are
 *               integer vectors) are contracted once per (q, -q) pair: the cosine rows of the pair form are even in q, the
 *               sine rows odd, C(+-q) = Ce +- Co.  The pairs are found on the device in every q_batch call (no host round
 *               trip; coordinates must match EXACTLY in binary, e.g. i/2^m meshes); lists with < 25 % of their q-points
 *               paired, the stacked forms and lists of < 256 q-points take the plain path.  0 (default) = off: the
 *               single-CTA pair search (24 us for 4096 q, 0.35 ms for 32768 q) costs more than the halved contraction
 *               saves at the sizes measured.  get_tuning("qfold_reps") = representatives of the
 *               LAST q_batch call if it took the fold, else 0 (synchronises the stream)
 *   "setk_pair" 1 (default) = the a1 GEMM of set_k_batch folds the +R / -R pairs of the Re list (real phases x complex sums
 *               g_W[e] +- g_W[ebar] formed on the fly: 2 instead of 3 tensor instructions per tile and k-step) whenever
 *               that saves time (batches of >= 12 k-points, where the three-multiply form is FP64-bound); 0 = always the
 *               three-multiply form.  get_tuning("setk_pair_rows") = ring rows (2 per pair) if the last set_k_batch used it
 *   "rot_plain" 1 = force the plain DFMA rotation kernel (the fallback for nmodes > 48)
 *   "rot_qg" / "rot_gb1" / "rot_mtw"   override the geometry of the tensor-core rotation kernel (rotate_v3.cuh):
 *               q-points per ring stage, b1 per C stage (forces the two-ring form), 8-row tiles of b2 per warp item
 *               (0 = automatic; measurement aids).  "rot_blk": how U_kq / ev reach shared memory: 0 = automatic,
 *               1 = one bulk copy per row into padded rows, 2 = one bulk copy per q-point at the natural pitch      */
int phoebe_elph_set_tuning(phoebe_elph_ctx* ctx, const char* key, int64_t value);
int phoebe_elph_get_tuning(const phoebe_elph_ctx* ctx, const char* key, int64_t* value);

int phoebe_elph_destroy(phoebe_elph_ctx* ctx);

/* Text of the last error on this context ("" if none); valid until the next call on ctx. */
const char* phoebe_elph_last_error(const phoebe_elph_ctx* ctx);

const char* phoebe_elph_version(void);

/* ---- Allocation-free variant of set_k (a1 + a2, Eq. 71) -------------------------------------------------
 * For callers that cannot allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
 * No context, no workspace: the Fourier-summed, not yet rotated tensor T[nRp][nw][nw][nmodes] (the scratch the context-based
 * path keeps in the caller's workspace) lives in a file-scope device array of PHOEBE_ELPH_NOALLOC_MAX_BYTES inside the
 * library -- every GPU that loads the library holds it until the process exits.  The call launches two kernels on
 * cuda_stream and returns without synchronising; it calls no cudaMalloc / cudaFree and no allocating library routine.
 *   gW_dev     DEVICE complex128 [nRp][nRe][nw][nw][nmodes], 16-B aligned (as in phoebe_elph_setup); read once
 *   Re_dev     DEVICE double [nRe][3] (crystal coordinates);  deg_e_dev DEVICE double [nRe] or NULL (= all 1)
 *   k_host     HOST double [3], read before the call returns
 *   Uk_dev     DEVICE complex128 [nw][nb1];  g1_out_dev DEVICE complex128 [nRp][nb1][nw][nmodes], written (caller-owned)
 * Conventions: those of a fresh context (phase_sign = +1, U_k not conjugated).
 * LIMIT: nRp * nw * nw * nmodes * 16 bytes <= PHOEBE_ELPH_NOALLOC_MAX_BYTES (e.g. the si-like cell: 343 * 8 * 8 * 6 * 16 =
 * 2.1 MB); larger problems are rejected with E_DIMS and a text that says so -- use phoebe_elph_set_k with a workspace.
 * SHARING: every call on a device uses the SAME array, which keeps the last call's contents (each call writes every element
 * before reading it, so nothing needs clearing); calls that overlap on the GPU (two streams, concurrently replayed graphs)
 * RACE on it: serialise them.
 * phoebe_elph_noalloc_setup(): looks up the array's device address for the CURRENT device (once per device; the first use
 * of a device may load the module): call it once per device before capturing; set_k_noalloc does the same lookup lazily.
 * Errors: E_NULL, E_DIMS, E_ALIGN, E_CUDA; text via phoebe_elph_noalloc_last_error() (per host thread). */
#define PHOEBE_ELPH_NOALLOC_MAX_BYTES (4u << 20)
int phoebe_elph_noalloc_setup(void);
int phoebe_elph_set_k_noalloc(const void* gW_dev, const double* Re_dev, const double* deg_e_dev, int32_t nRe, int32_t nRp,
                              int32_t nw, int32_t nmodes, int32_t nb1, const double* k_host, const void* Uk_dev,
                              void* g1_out_dev, void* cuda_stream);
const char* phoebe_elph_noalloc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* PHOEBE_ELPH_H */
