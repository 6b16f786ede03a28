/*
 * oracle_elph.c -- CPU ORACLE for the el-ph Wannier->Bloch |g|^2 hot path.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call this.  It shares
 * no code, header, table or helper with the CUDA path under
 * paper_2111_14999_b200/csrc and neither side includes the other.
 *
 * Plain, slow, obviously-correct C99 (double complex, nested loops), written
 * from /root/reference/PAPER.md:
 *
 *   Eq. 13  g0(k,q) = sum_{Re,Rp} e^{ik.Re + iq.Rp}
 *                                      U_{k+q} g0(Re,Rp) U_k^dagger z_q
 *   Eq. 7   g = (1/(2 m omega_{q nu}))^{1/2} g0 ;  b <-> k (ket),
 *                           b' <-> k+q (bra)
 *   Eq. 11  columns of U_k are the eigenvectors
 *   Eq. 70/71 (L564-L570)   the factorisation: fixed-k precompute (set_k),
 *                           then completion per k' (q_batch)
 *
 * Readings of the garbled / silent points:
 *   R1  phase = exp(+2*pi*i * k.R), k,q fractional (crystal) coords, L510
 *   R2  every term divided by deg_e[e]*deg_p[p] (Wigner-Seitz weights)
 *   R3  U_k plain on the k (ket) index, conj(U_kq) on the k+q (bra) index
 *   R5  g_W[p][e][w1][w2][kappa]: w1 <-> k / U_k / b1,  w2 <-> k+q / U_kq / b2
 *   R6  ev[q][kappa][nu] used unconjugated; masses folded into ev by the caller
 *   R7  out = 0 where omega <= 0
 *
 * Definition computed (exact; the factorised form reaches the same number):
 *
 *   G(k,q)[b1][b2][nu] = sum_e sum_p (e^{2 pi i k.Re_e}/deg_e[e]) (e^{2 pi i q.Rp_p}/deg_p[p])
 *        sum_{w1,w2,kappa} U_k[w1][b1] conj(U_kq[w2][b2]) ev[kappa][nu] g_W[p][e][w1][w2][kappa]
 *   out[q][b1][b2][nu] = |G|^2 / (2 omega[q][nu])
 *
 * Layouts: all arrays C-order; complex = (re, im) pairs of doubles.
 *   g_W [nRp][nRe][nw][nw][nm]   Re [nRe][3]  Rp [nRp][3]  deg_e [nRe]  deg_p [nRp]
 *   U_k [nw][nb1]   U_kq [nq][nw][nb2]   ev [nq][nm][nm]   omega [nq][nm]
 *   g1  [nRp][nb1][nw][nm]      out [nq][nb1][nb2][nm] (double)
 *
 * Parity pins: tests/test_oracle_pins.py (P1..P12 of SURVEY 8(c)); nothing
 * here is "parity unpinned".
 */
#include <complex.h>
#include <math.h>
#include <stddef.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

static const double ORACLE_PI = 3.14159265358979323846264338327950288;

/* e^{2 pi i k.R}: the integer part of x = k.R is dropped first (exact
 * subtraction; e^{2 pi i n} = 1), then cos/sin of 2*pi*frac.  Reading R1. */
static cplx oracle_phase(const double *k, const double *R)
{
    double x = k[0] * R[0] + k[1] * R[1] + k[2] * R[2];
    x -= round(x);
    return cos(2.0 * ORACLE_PI * x) + I * sin(2.0 * ORACLE_PI * x);
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------
 * oracle_direct: Eq. 13 + Eq. 7 written out as the plain double sum over
 * (Re, Rp) with all three rotations inside -- nothing factorised, nothing
 * precomputed.  Accumulates in long double.  Tiny inputs only.
 * ---------------------------------------------------------------------- */
int oracle_direct(int nRe, int nRp, int nw, int nm, int nb1, int nb2, int nq,
                  const cplx *gW, const double *Re, const double *Rp,
                  const double *deg_e, const double *deg_p,
                  const double *k, const cplx *Uk,
                  const double *q, const cplx *Ukq, const cplx *ev,
                  const double *omega, double *out)
{
    for (int iq = 0; iq < nq; ++iq)
        for (int b1 = 0; b1 < nb1; ++b1)
            for (int b2 = 0; b2 < nb2; ++b2)
                for (int nu = 0; nu < nm; ++nu) {
                    long double complex G = 0.0L;
                    for (int e = 0; e < nRe; ++e) {
                        cplx phe = oracle_phase(k, Re + 3 * e) / (deg_e ? deg_e[e] : 1.0);
                        for (int p = 0; p < nRp; ++p) {
                            cplx php = oracle_phase(q + 3 * iq, Rp + 3 * p) / (deg_p ? deg_p[p] : 1.0);
                            long double complex s = 0.0L;
                            for (int w1 = 0; w1 < nw; ++w1)
                                for (int w2 = 0; w2 < nw; ++w2)
                                    for (int ka = 0; ka < nm; ++ka) {
                                        cplx g = gW[((((size_t)p * nRe + e) * nw + w1) * nw + w2) * nm + ka];
                                        cplx u1 = Uk[(size_t)w1 * nb1 + b1];
                                        cplx u2 = conj(Ukq[((size_t)iq * nw + w2) * nb2 + b2]);
                                        cplx z = ev[((size_t)iq * nm + ka) * nm + nu];
                                        s += (long double complex)(u1 * u2) * (long double complex)(z * g);
                                    }
                            G += (long double complex)(phe * php) * s;
                        }
                    }
                    double w = omega[(size_t)iq * nm + nu];
                    long double m2 = creall(G) * creall(G) + cimagl(G) * cimagl(G);
                    out[(((size_t)iq * nb1 + b1) * nb2 + b2) * nm + nu] =
                        (w > 0.0) ? (double)(m2 / (2.0L * (long double)w)) : 0.0;
                }
    return 0;
}

/* ------------------------------------------------------------------------
 * oracle_setk_slab: Eq. 71 for ONE phonon lattice vector p (steps a1, a2).
 *   T[w1][w2][ka]   = sum_e (e^{2 pi i k.Re_e}/deg_e[e]) gW_p[e][w1][w2][ka]
 *   g1_p[b1][w2][ka] = sum_{w1} U_k[w1][b1] T[w1][w2][ka]
 * gW_p is the slab [nRe][nw][nw][nm]; g1_p is [nb1][nw][nm].
 * ---------------------------------------------------------------------- */
int oracle_setk_slab(int nRe, int nw, int nm, int nb1,
                     const cplx *gW_p, const double *Re, const double *deg_e,
                     const double *k, const cplx *Uk, cplx *g1_p)
{
    size_t X = (size_t)nw * nw * nm;
    cplx *T = (cplx *)calloc(X, sizeof(cplx));
    if (!T) return -1;
    for (int e = 0; e < nRe; ++e) {
        cplx ph = oracle_phase(k, Re + 3 * e) / (deg_e ? deg_e[e] : 1.0);
        const cplx *g = gW_p + (size_t)e * X;
        for (size_t x = 0; x < X; ++x) T[x] += ph * g[x];
    }
    for (int b1 = 0; b1 < nb1; ++b1)
        for (int w2 = 0; w2 < nw; ++w2)
            for (int ka = 0; ka < nm; ++ka) {
                cplx s = 0.0;
                for (int w1 = 0; w1 < nw; ++w1)
                    s += Uk[(size_t)w1 * nb1 + b1] * T[((size_t)w1 * nw + w2) * nm + ka];
                g1_p[((size_t)b1 * nw + w2) * nm + ka] = s;
            }
    free(T);
    return 0;
}

/* oracle_setk: Eq. 71 for all p (g_W fully resident on the host). */
int oracle_setk(int nRe, int nRp, int nw, int nm, int nb1,
                const cplx *gW, const double *Re, const double *deg_e,
                const double *k, const cplx *Uk, cplx *g1)
{
    size_t slab = (size_t)nRe * nw * nw * nm, N = (size_t)nb1 * nw * nm;
    int rc = 0;
#pragma omp parallel for schedule(static)
    for (int p = 0; p < nRp; ++p) {
        int r = oracle_setk_slab(nRe, nw, nm, nb1, gW + (size_t)p * slab, Re, deg_e, k, Uk,
                                 g1 + (size_t)p * N);
        if (r) rc = r;
    }
    return rc;
}

/* ------------------------------------------------------------------------
 * oracle_qbatch: the rest of Eq. 70 + Eq. 7 (steps a3..a7), one q at a time.
 *   C[b1][w2][ka]  = sum_p (e^{2 pi i q.Rp_p}/deg_p[p]) g1[p][b1][w2][ka]
 *   D[b1][b2][ka]  = sum_{w2} conj(U_kq[w2][b2]) C[b1][w2][ka]
 *   E[b1][b2][nu]  = sum_{ka} D[b1][b2][ka] ev[ka][nu]
 *   out            = |E|^2 / (2 omega[nu])          (0 where omega <= 0)
 * OpenMP over q only (used when the oracle is timed as the CPU baseline).
 * ---------------------------------------------------------------------- */
int oracle_qbatch(int nRp, int nw, int nm, int nb1, int nb2, int nq,
                  const cplx *g1, const double *Rp, const double *deg_p,
                  const double *q, const cplx *Ukq, const cplx *ev,
                  const double *omega, double *out)
{
    size_t N = (size_t)nb1 * nw * nm;
    int rc = 0;
#pragma omp parallel for schedule(static)
    for (int iq = 0; iq < nq; ++iq) {
        cplx *C = (cplx *)calloc(N, sizeof(cplx));
        cplx *D = (cplx *)malloc((size_t)nb1 * nb2 * nm * sizeof(cplx));
        if (!C || !D) { rc = -1; free(C); free(D); continue; }
        for (int p = 0; p < nRp; ++p) {
            cplx ph = oracle_phase(q + 3 * iq, Rp + 3 * p) / (deg_p ? deg_p[p] : 1.0);
            const cplx *g = g1 + (size_t)p * N;
            for (size_t n = 0; n < N; ++n) C[n] += ph * g[n];
        }
        const cplx *U = Ukq + (size_t)iq * nw * nb2;
        const cplx *Z = ev + (size_t)iq * nm * nm;
        for (int b1 = 0; b1 < nb1; ++b1)
            for (int b2 = 0; b2 < nb2; ++b2)
                for (int ka = 0; ka < nm; ++ka) {
                    cplx s = 0.0;
                    for (int w2 = 0; w2 < nw; ++w2)
                        s += conj(U[(size_t)w2 * nb2 + b2]) * C[((size_t)b1 * nw + w2) * nm + ka];
                    D[((size_t)b1 * nb2 + b2) * nm + ka] = s;
                }
        for (int b1 = 0; b1 < nb1; ++b1)
            for (int b2 = 0; b2 < nb2; ++b2)
                for (int nu = 0; nu < nm; ++nu) {
                    cplx s = 0.0;
                    for (int ka = 0; ka < nm; ++ka)
                        s += D[((size_t)b1 * nb2 + b2) * nm + ka] * Z[(size_t)ka * nm + nu];
                    double w = omega[(size_t)iq * nm + nu];
                    double m2 = creal(s) * creal(s) + cimag(s) * cimag(s);
                    out[(((size_t)iq * nb1 + b1) * nb2 + b2) * nm + nu] = (w > 0.0) ? m2 / (2.0 * w) : 0.0;
                }
        free(C);
        free(D);
    }
    return rc;
}

/* ========================================================================
 * electron linewidths from |g|^2 (Eq. 29)
 * with the Gaussian approximation of the Dirac delta (Eq. 61).
 *
 *   1/tau_{k b} = (2 pi / (N_k V)) sum_{k' b' q nu} |g_{b b' nu}(k,k')|^2
 *        [ (1 - f_{k'b'} + n_{q nu}) delta(eps_{kb} - hbar omega_{q nu} - eps_{k'b'})
 *        + (    f_{k'b'} + n_{q nu}) delta(eps_{kb} + hbar omega_{q nu} - eps_{k'b'}) ] delta(k - k' + q)
 *   delta(x) ~ exp(-x^2 / sigma^2) / (sqrt(pi) sigma)                              (Eq. 61)
 *   f(eps) = 1 / (e^{(eps - mu)/k_B T} + 1)   (L212),   n(omega) = 1 / (e^{omega/k_B T} - 1)
 *
 * Readings (R16-R18):
 *   R16 delta(k - k' + q) selects k' = k + q: the sum runs over the q list only; b = b1 (band at k),
 *       b' = b2 (band at k+q), so |g_{b b' nu}|^2 = out[q][b1][b2][nu] of Eq. 7/13.
 *   R17 the prefactor 2 pi/(N_k V) (and any unit conversion) is the caller's `pref`; hbar = 1 (R8).
 *   R18 modes with omega <= 0 contribute nothing (their |g|^2 is 0 by R7; n is not evaluated).
 *
 *   rate[b1] += pref * sum_{q, b2, nu} out[q][b1][b2][nu] * W(eps_k[b1], eps_kq[q][b2], omega[q][nu])
 *
 * Plain loops, long double accumulation.
 * ====================================================================== */
double oracle_fermi(double eps, double mu, double kT) { return 1.0 / (exp((eps - mu) / kT) + 1.0); }

double oracle_bose(double omega, double kT) { return 1.0 / (exp(omega / kT) - 1.0); }

double oracle_delta_gauss(double x, double sigma)
{
    return exp(-(x * x) / (sigma * sigma)) / (sqrt(ORACLE_PI) * sigma);
}

/* the square bracket of Eq. 29 for one (b, b', nu) term */
double oracle_rate_weight(double eps_kb, double eps_kqb, double omega, double kT, double mu, double sigma)
{
    if (!(omega > 0.0)) return 0.0;
    double f = oracle_fermi(eps_kqb, mu, kT), n = oracle_bose(omega, kT);
    return (1.0 - f + n) * oracle_delta_gauss(eps_kb - omega - eps_kqb, sigma) +
           (f + n) * oracle_delta_gauss(eps_kb + omega - eps_kqb, sigma);
}

int oracle_rates(int nq, int nb1, int nb2, int nm, const double *out /* [nq][nb1][nb2][nm] */,
                 const double *eps_k /* [nb1] */, const double *eps_kq /* [nq][nb2] */,
                 const double *omega /* [nq][nm] */, double kT, double mu, double sigma, double pref,
                 double *rate /* [nb1], accumulated into */)
{
    for (int b1 = 0; b1 < nb1; ++b1) {
        long double s = 0.0L;
        for (int iq = 0; iq < nq; ++iq)
            for (int b2 = 0; b2 < nb2; ++b2)
                for (int nu = 0; nu < nm; ++nu) {
                    double w = oracle_rate_weight(eps_k[b1], eps_kq[(size_t)iq * nb2 + b2],
                                                  omega[(size_t)iq * nm + nu], kT, mu, sigma);
                    s += (long double)out[(((size_t)iq * nb1 + b1) * nb2 + b2) * nm + nu] * (long double)w;
                }
        rate[b1] += (double)((long double)pref * s);
    }
    return 0;
}

/* ========================================================================
 * polar (long-range) correction, Eq. 14-15 (L139-L147):
 *
 *   g = g^S + g^L                                                               (Eq. 14)
 *   g^L_{b'b nu}(k,q) = i (4 pi / V)(e^2 / 4 pi eps0) sum_s (hbar / (2 N_q m_s omega_{q nu}))^{1/2}
 *        sum_{G != -q} [(q+G).Z*_s.z^s_{q nu}] / [(q+G).eps_inf.(q+G)]
 *        <psi_{k+q,b'}| e^{i(q+G).r} |psi_{k,b}>                                 (Eq. 15)
 *
 * Readings (R20-R24):
 *   R20 the matrix element is taken in the Wannier-gauge approximation of the paper's Ref. [34]:
 *       <psi_{k+q,b'}|e^{i(q+G).r}|psi_{k,b}> = [U_{k+q}^dagger U_k]_{b'b}  (Eq. 15 prints psi_{k+q} on both
 *       sides; the ket belongs to k as in Eq. 7);  O[b1][b2] = sum_w conj(U_kq[w][b2]) U_k[w][b1].
 *   R21 (hbar/(2 m_s omega))^{1/2}: 1/sqrt(m_s) is folded into ev by the caller (R6), 1/sqrt(2 omega) is the
 *       library's final 1/(2 omega) on |.|^2 exactly as for the short-range part (R7: 0 where omega <= 0),
 *       1/sqrt(N_q) and (4 pi/V)(e^2/4 pi eps0) are the caller's real `coeff`.  So what is ADDED to the
 *       amplitude E of Eq. 13 before |.|^2 is   L[q][b1][b2][nu] = P[q][nu] O[q][b1][b2],
 *         P[q][nu] = i coeff sum_G [Q.Zeff_nu] / [Q.eps_inf.Q],   Q = (q+G) in Cartesian coordinates,
 *         Zeff_nu[a] = sum_s sum_b Z*_s[a][b] ev[q][3s+b][nu].
 *   R22 q, G are in crystal coordinates (L510); Q = (q+G)_0 B[0] + (q+G)_1 B[1] + (q+G)_2 B[2] with the rows
 *       of `recip` = reciprocal lattice vectors (any 2 pi inside them).
 *   R23 "G != -q": a term is skipped when, and only when, Q is exactly the zero vector.  The sum runs over the
 *       caller's finite list of G (Eq. 15 prints no convergence factor; none is applied).
 *   R24 (q+G).Z*_s.z = sum_{a,b} Q_a Z*_s[a][b] z_b  (row index of Z* with the wavevector).
 *
 * Plain loops.  Pins: tests/test_oracle_polar_pins.py (PP1-PP8).
 * ====================================================================== */
int oracle_polar_amplitude(int nq, int nm, int nG, const double *q /* [nq][3] */, const cplx *ev /* [nq][nm][nm] */,
                           const double *recip /* [3][3] */, const double *G /* [nG][3] */,
                           const double *Zstar /* [nm/3][3][3] */, const double *eps_inf /* [3][3] */, double coeff,
                           cplx *P /* [nq][nm] */)
{
    if (nm % 3) return -2;
    int nat = nm / 3;
    for (int iq = 0; iq < nq; ++iq)
        for (int nu = 0; nu < nm; ++nu) {
            cplx zeff[3] = {0.0, 0.0, 0.0};
            for (int s = 0; s < nat; ++s)
                for (int a = 0; a < 3; ++a)
                    for (int b = 0; b < 3; ++b)
                        zeff[a] += Zstar[(s * 3 + a) * 3 + b] * ev[((size_t)iq * nm + 3 * s + b) * nm + nu];
            cplx sum = 0.0;
            for (int ig = 0; ig < nG; ++ig) {
                double c[3], Q[3];
                for (int a = 0; a < 3; ++a) c[a] = q[3 * iq + a] + G[3 * ig + a];
                for (int a = 0; a < 3; ++a) Q[a] = c[0] * recip[a] + c[1] * recip[3 + a] + c[2] * recip[6 + a];
                if (Q[0] == 0.0 && Q[1] == 0.0 && Q[2] == 0.0) continue;       /* G = -q */
                double den = 0.0;
                for (int a = 0; a < 3; ++a)
                    for (int b = 0; b < 3; ++b) den += Q[a] * eps_inf[a * 3 + b] * Q[b];
                cplx num = Q[0] * zeff[0] + Q[1] * zeff[1] + Q[2] * zeff[2];
                sum += num / den;
            }
            P[(size_t)iq * nm + nu] = I * coeff * sum;
        }
    return 0;
}

/* oracle_qbatch with the long-range amplitude added before |.|^2 (Eq. 14):
 *   E[b1][b2][nu] = (short-range E of oracle_qbatch) + P[q][nu] * sum_w conj(U_kq[w][b2]) U_k[w][b1] */
int oracle_qbatch_polar(int nRp, int nw, int nm, int nb1, int nb2, int nq,
                        const cplx *g1, const double *Rp, const double *deg_p,
                        const double *q, const cplx *Ukq, const cplx *ev, const double *omega,
                        const cplx *Uk /* [nw][nb1] */, const cplx *P /* [nq][nm] */, double *out)
{
    size_t N = (size_t)nb1 * nw * nm;
    int rc = 0;
#pragma omp parallel for schedule(static)
    for (int iq = 0; iq < nq; ++iq) {
        cplx *C = (cplx *)calloc(N, sizeof(cplx));
        if (!C) { rc = -1; continue; }
        for (int p = 0; p < nRp; ++p) {
            cplx ph = oracle_phase(q + 3 * iq, Rp + 3 * p) / (deg_p ? deg_p[p] : 1.0);
            const cplx *g = g1 + (size_t)p * N;
            for (size_t n = 0; n < N; ++n) C[n] += ph * g[n];
        }
        const cplx *U = Ukq + (size_t)iq * nw * nb2;
        const cplx *Z = ev + (size_t)iq * nm * nm;
        for (int b1 = 0; b1 < nb1; ++b1)
            for (int b2 = 0; b2 < nb2; ++b2) {
                cplx ov = 0.0;                                   /* [U_kq^dagger U_k]_{b2 b1} */
                for (int w = 0; w < nw; ++w) ov += conj(U[(size_t)w * nb2 + b2]) * Uk[(size_t)w * nb1 + b1];
                for (int nu = 0; nu < nm; ++nu) {
                    cplx s = 0.0;
                    for (int ka = 0; ka < nm; ++ka)
                        for (int w2 = 0; w2 < nw; ++w2)
                            s += conj(U[(size_t)w2 * nb2 + b2]) * C[((size_t)b1 * nw + w2) * nm + ka] *
                                 Z[(size_t)ka * nm + nu];
                    s += P[(size_t)iq * nm + nu] * ov;
                    double w = omega[(size_t)iq * nm + nu];
                    double m2 = creal(s) * creal(s) + cimag(s) * cimag(s);
                    out[(((size_t)iq * nb1 + b1) * nb2 + b2) * nm + nu] = (w > 0.0) ? m2 / (2.0 * w) : 0.0;
                }
            }
        free(C);
    }
    return rc;
}

/* ========================================================================
 * SURVEY 8(f) f4 (second half) -- three-phonon coupling, Eq. 5 (L82), the second workload with the
 * Eq. 70 shape (L137: "Eq. 5 and Eq. 13 are similar from a mathematical point of view"):
 *
 *   V3(q nu, q' nu', q'' nu'') = (1/N0^3)(2/hbar)^{3/2} sum_{R R'} sum_{a b c} [mass / frequency factor]
 *        z*_{q nu}[a] z*_{q' nu'}[b] z*_{q'' nu''}[c] e^{-i(q.R + q'.R')} V3(a R, b R', c 0)
 *
 * Readings (R25-R27):
 *   R25 the mass / frequency factor is printed as sqrt(m m' m'' / (omega omega' omega'')) (masses upstairs,
 *       garbled); whatever it is, it factorises over the three phonons, so -- like 1/sqrt(m) in R6 -- it is
 *       folded into the three eigenvector arrays by the caller, as is the constant prefactor.  The oracle (and
 *       the library) compute the bare triple contraction and return its squared modulus.
 *   R26 Eq. 5 prints z_{q' nu'}^{s'' beta}: the atom index of the second eigenvector is s' (the one V3 carries
 *       with beta).
 *   R27 all three eigenvectors are conjugated and both phases carry a MINUS sign, e^{-2 pi i (q.R + q'.R')} with
 *       q, q' in crystal coordinates (L510) -- the opposite of Eq. 13's sign.
 *
 *   out[nu][nu'][nu''] = | sum_{R,R'} e^{-2 pi i q.R} e^{-2 pi i q'.R'}
 *                          sum_{a,b,c} conj(z[a][nu]) conj(z1[b][nu']) conj(z2[c][nu'']) V3[R'][R][a][b][c] |^2
 *
 * Layout: V3 [nR2][nR][nm][nm][nm] (R' slowest, as g_W's [Rp][Re]); z [nm][n0], z1 [nq][nm][n1], z2 [nq][nm][nm];
 * q [3]; q1 [nq][3]; out [nq][n0][n1][nm].  Plain 7-deep loop, long double accumulation.
 * Pins: tests/test_oracle_v3_pins.py (VP1-VP4).
 * ====================================================================== */
int oracle_v3sq(int nR, int nR2, int nm, int n0, int n1, int nq, const cplx *V3, const double *R, const double *R2,
                const double *q, const cplx *z, const double *q1, const cplx *z1, const cplx *z2, double *out)
{
#pragma omp parallel for schedule(static)
    for (int iq = 0; iq < nq; ++iq)
        for (int nu = 0; nu < n0; ++nu)
            for (int nu1 = 0; nu1 < n1; ++nu1)
                for (int nu2 = 0; nu2 < nm; ++nu2) {
                    long double sr = 0.0L, si = 0.0L;
                    for (int r2 = 0; r2 < nR2; ++r2)
                        for (int r = 0; r < nR; ++r) {
                            cplx ph = conj(oracle_phase(q, R + 3 * r)) * conj(oracle_phase(q1 + 3 * iq, R2 + 3 * r2));
                            cplx s = 0.0;
                            for (int a = 0; a < nm; ++a)
                                for (int b = 0; b < nm; ++b)
                                    for (int c = 0; c < nm; ++c)
                                        s += conj(z[(size_t)a * n0 + nu]) * conj(z1[((size_t)iq * nm + b) * n1 + nu1]) *
                                             conj(z2[((size_t)iq * nm + c) * nm + nu2]) *
                                             V3[((((size_t)r2 * nR + r) * nm + a) * nm + b) * nm + c];
                            s *= ph;
                            sr += creal(s); si += cimag(s);
                        }
                    out[(((size_t)iq * n0 + nu) * n1 + nu1) * nm + nu2] = (double)(sr * sr + si * si);
                }
    return 0;
}
