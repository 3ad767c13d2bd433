/*
 * nmso.c -- fp64 CPU ORACLE for the direct-summation SANS core of
 * arxiv/paper_2601_18444 (NuMagSANS).  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference leg may call this file.  It shares no code, header,
 * table or helper with the CUDA path in paper_2601_18444_b200/ and the
 * product path never routes through it.
 *
 * Every function is the plain definition from PAPER.md written out in
 * fp64 with libm sin/cos, parallel over detector points only (OpenMP);
 * no blocking, no fusion, no reordering beyond the equations.  Citations
 * "Lnnn" are line numbers of /root/reference/PAPER.md.  Readings of
 * silent / garbled passages are the ones listed in DESIGN.md section 3.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): dimer closed form,
 * F(0) = sum w, Dirichlet-kernel product for a cuboid lattice,
 * translation invariance, rotate-sample == rotate-q, brute force in
 * Python complex arithmetic, Q.q = 0, channel sum rules, expanded forms
 * Eq. 9/15/28, uniform-m angular factors Eq. 60-63, Table II I(0)
 * values, sphere form factor, azimuthal means Eq. 65-67, Fourier-Bessel
 * of the sphere form factor (gamma_0), form/interference split of two
 * identical particles, angular modal decomposition of trigonometric maps
 * (A_0^c / A_2^c = -1 for sin^2, A_0^c / A_4^c = -1 for sin^2 cos^2, L199),
 * 2-D correlation of a ring (2 pi J0, -2 pi J2 cos 2 alpha), of a Gaussian,
 * parity symmetries and brute force.
 * No function here is "parity unpinned".
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC -o libnmso.so nmso.c -lm
 */
#define _GNU_SOURCE
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define NMSO_OK 0
#define NMSO_E_ARG 1
#define NMSO_E_NOMEM 2

/* response kinds, same order as include/nms.h (the numbering is part of the ABI, not shared code) */
enum { K_NUC = 0, K_MAG, K_UNPOL, K_PROJ, K_NM, K_SF, K_CHI, K_PM, K_MP, K_PP, K_MM, K_POL_PLUS, K_POL_MINUS, K_COUNT };

int nmso_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------
 * Rotated laboratory-frame coordinates and moments.
 * Eq. 38-40 (L331-L339): (X,Y,Z) = R (x^{kl} + r^k); r^k = 0 when no
 * StructData is given (L341).  The moment is rotated with the sample,
 * m' = R m (reading 2; north_star: M~ = sum (R m_j) e^{-i q.R r_j}).
 * pos, m: float32 inputs promoted to fp64; all products in fp64.
 * part_of_cell is derived from offsets[K+1] (L310-L317).
 * ---------------------------------------------------------------------- */
static int rotate_sample(const float *pos, const float *m, int64_t W,
                         const int64_t *offsets, int64_t K, const float *centres,
                         const double *R, double *rp /*[W][3]*/, double *rm /*[W][3] or NULL*/)
{
    static const double I3[9] = {1, 0, 0, 0, 1, 0, 0, 0, 1};
    if (!R) R = I3;
    if (centres && (!offsets || K <= 0)) return NMSO_E_ARG;
    int64_t k = 0;
    for (int64_t j = 0; j < W; ++j) {
        double x = pos[3 * j + 0], y = pos[3 * j + 1], z = pos[3 * j + 2];
        if (centres) {
            while (k + 1 < K && j >= offsets[k + 1]) ++k;
            x += (double)centres[3 * k + 0];
            y += (double)centres[3 * k + 1];
            z += (double)centres[3 * k + 2];
        }
        rp[3 * j + 0] = R[0] * x + R[1] * y + R[2] * z;   /* Eq. 38 */
        rp[3 * j + 1] = R[3] * x + R[4] * y + R[5] * z;   /* Eq. 39 */
        rp[3 * j + 2] = R[6] * x + R[7] * y + R[8] * z;   /* Eq. 40 */
        if (rm) {
            double mx = m[3 * j + 0], my = m[3 * j + 1], mz = m[3 * j + 2];
            rm[3 * j + 0] = R[0] * mx + R[1] * my + R[2] * mz;
            rm[3 * j + 1] = R[3] * mx + R[4] * my + R[5] * mz;
            rm[3 * j + 2] = R[6] * mx + R[7] * my + R[8] * mz;
        }
    }
    return NMSO_OK;
}

/* ------------------------------------------------------------------------
 * Detector points.  Eq. 6 (L58): q^ = (0, sin th, cos th); L343: q_y = q sin th,
 * q_z = q cos th.  The float32 abscissae are promoted to fp64 first.
 *  type 0 polar     : u0 = |q| [n0], u1 = theta [n1]
 *  type 1 cartesian : u0 = q_z [n0], u1 = q_y [n1]; theta = atan2(q_y, q_z), atan2(0,0) = 0
 *  type 2 list      : u0 = q_y [n0], u1 = q_z [n0], n1 = 1
 * flat index = i0 * n1 + i1.
 * ---------------------------------------------------------------------- */
int nmso_grid_points(int type, int n0, int n1, const float *u0, const float *u1,
                     double *qy, double *qz, double *theta)
{
    if (n0 <= 0 || n1 <= 0 || !u0 || !u1) return NMSO_E_ARG;
    for (int i0 = 0; i0 < n0; ++i0)
        for (int i1 = 0; i1 < n1; ++i1) {
            int64_t f = (int64_t)i0 * n1 + i1;
            if (type == 0) {
                double q = u0[i0], th = u1[i1];
                qy[f] = q * sin(th);
                qz[f] = q * cos(th);
                theta[f] = th;
            } else if (type == 1) {
                qz[f] = u0[i0];
                qy[f] = u1[i1];
                theta[f] = atan2(qy[f], qz[f]);
            } else if (type == 2) {
                qy[f] = u0[i0];
                qz[f] = u1[i0];
                theta[f] = atan2(qy[f], qz[f]);
            } else
                return NMSO_E_ARG;
        }
    return NMSO_OK;
}

/* ------------------------------------------------------------------------
 * Direct sums, Eq. 42-47 (L353-L368) without any normalisation prefactor
 * (reading 4: raw sums):
 *     A_c(q) = sum_j w_{c,j} exp(-i q . r'_j),   c in {N, x, y, z}
 *     Re A_c = + sum w cos(Psi)   (Eq. 44, 46)
 *     Im A_c = - sum w sin(Psi)   (Eq. 45, 47)
 *     Psi_j  = q_x X_j + q_y Y_j + q_z Z_j;  on the detector q_x = 0 (Eq. 41).
 * qx may be NULL (= 0).  The 3-D entry point exists for the rotation pin
 * (rotating the sample by R == rotating q by R^T).
 * out: [8][nq] planes Re N, Im N, Re Mx, Im Mx, Re My, Im My, Re Mz, Im Mz.
 * wsum (optional, [4]): sum_j |w_{c,j}| of the rotated weights (tolerance denominators).
 * ---------------------------------------------------------------------- */
int nmso_amplitudes(const float *pos, const float *N, const float *m, int64_t W,
                    const int64_t *offsets, int64_t K, const float *centres, const double *R,
                    const double *qx, const double *qy, const double *qz, int64_t nq,
                    double *out, double *wsum)
{
    if (!pos || W <= 0 || nq <= 0 || !qy || !qz || !out) return NMSO_E_ARG;
    double *rp = (double *)malloc(sizeof(double) * 3 * (size_t)W);
    double *rm = m ? (double *)malloc(sizeof(double) * 3 * (size_t)W) : NULL;
    if (!rp || (m && !rm)) { free(rp); free(rm); return NMSO_E_NOMEM; }
    int rc = rotate_sample(pos, m, W, offsets, K, centres, R, rp, rm);
    if (rc) { free(rp); free(rm); return rc; }
    if (wsum) {
        wsum[0] = wsum[1] = wsum[2] = wsum[3] = 0.0;
        for (int64_t j = 0; j < W; ++j) {
            if (N) wsum[0] += fabs((double)N[j]);
            if (rm) { wsum[1] += fabs(rm[3 * j]); wsum[2] += fabs(rm[3 * j + 1]); wsum[3] += fabs(rm[3 * j + 2]); }
        }
    }
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t i = 0; i < nq; ++i) {
        const double kx = qx ? qx[i] : 0.0, ky = qy[i], kz = qz[i];
        double aN = 0, bN = 0, ax = 0, bx = 0, ay = 0, by = 0, az = 0, bz = 0;
        for (int64_t j = 0; j < W; ++j) {
            const double psi = kx * rp[3 * j] + ky * rp[3 * j + 1] + kz * rp[3 * j + 2];
            const double c = cos(psi), s = sin(psi);
            if (N) { const double w = N[j]; aN += w * c; bN -= w * s; }
            if (rm) {
                ax += rm[3 * j] * c;     bx -= rm[3 * j] * s;
                ay += rm[3 * j + 1] * c; by -= rm[3 * j + 1] * s;
                az += rm[3 * j + 2] * c; bz -= rm[3 * j + 2] * s;
            }
        }
        out[0 * nq + i] = aN; out[1 * nq + i] = bN;
        out[2 * nq + i] = ax; out[3 * nq + i] = bx;
        out[4 * nq + i] = ay; out[5 * nq + i] = by;
        out[6 * nq + i] = az; out[7 * nq + i] = bz;
    }
    free(rp); free(rm);
    return NMSO_OK;
}

/* ------------------------------------------------------------------------
 * Response functions at one detector point, Section II (L35-L174).
 * Inputs: the four complex amplitudes (already scaled by sN, sM), theta,
 * unit polarisation P.  Coded from the VECTOR definitions:
 *   q^ = (0, sin th, cos th)                               Eq. 6  L58
 *   Q  = q^ x (q^ x M~)                                    Eq. 5  L54
 *   NUC = |N~|^2                                           Eq. 3  L48
 *   MAG = |Q|^2                                            Eq. 4  L50
 *   PROJ = |P.Q|^2                                         Eq. 8  L66
 *   SF  = MAG - PROJ                                       Eq. 13
 *   CHI = -i P.(Q x Q*)                                    Eq. 14
 *   PM  = SF + CHI, MP = SF - CHI                          Eq. 11-12
 *   NM  = P.(N~ Q* + N~* Q)                                Eq. 18
 *   PP  = NUC + NM + PROJ, MM = NUC - NM + PROJ            Eq. 16-17
 *   POL+ = PP + PM, POL- = MM + MP                         Eq. 23-24
 *   UNPOL = (PP + MM + PM + MP)/2                          Eq. 27
 * The common prefactor 8 pi^3 / V and b_H are carried by invV, sN, sM
 * (reading 4).
 * ---------------------------------------------------------------------- */
static void cross3(const double complex a[3], const double complex b[3], double complex o[3])
{
    o[0] = a[1] * b[2] - a[2] * b[1];
    o[1] = a[2] * b[0] - a[0] * b[2];
    o[2] = a[0] * b[1] - a[1] * b[0];
}

static void responses_at_point(double complex An, const double complex M[3], double theta,
                               const double P[3], double invV, double val[K_COUNT])
{
    const double complex qh[3] = {0.0, sin(theta), cos(theta)};
    double complex t[3], Q[3], Qc[3], QxQc[3];
    cross3(qh, M, t);
    cross3(qh, t, Q);                                   /* Eq. 5 */
    for (int a = 0; a < 3; ++a) Qc[a] = conj(Q[a]);
    cross3(Q, Qc, QxQc);
    const double complex PQ = P[0] * Q[0] + P[1] * Q[1] + P[2] * Q[2];
    const double nuc = creal(An * conj(An));
    const double mag = creal(Q[0] * Qc[0] + Q[1] * Qc[1] + Q[2] * Qc[2]);
    const double proj = creal(PQ * conj(PQ));
    const double complex chi_c = -I * (P[0] * QxQc[0] + P[1] * QxQc[1] + P[2] * QxQc[2]);
    const double chi = creal(chi_c);                    /* Q x Q* is purely imaginary */
    double complex nm_c = 0;
    for (int a = 0; a < 3; ++a) nm_c += P[a] * (An * Qc[a] + conj(An) * Q[a]);
    const double nm = creal(nm_c);
    const double sf = mag - proj;
    const double pm = sf + chi, mp = sf - chi;
    const double pp = nuc + nm + proj, mm = nuc - nm + proj;
    val[K_NUC] = invV * nuc;   val[K_MAG] = invV * mag;   val[K_PROJ] = invV * proj;
    val[K_NM] = invV * nm;     val[K_SF] = invV * sf;     val[K_CHI] = invV * chi;
    val[K_PM] = invV * pm;     val[K_MP] = invV * mp;     val[K_PP] = invV * pp;     val[K_MM] = invV * mm;
    val[K_POL_PLUS] = invV * (pp + pm);
    val[K_POL_MINUS] = invV * (mm + mp);
    val[K_UNPOL] = invV * 0.5 * (pp + mm + pm + mp);
}

static int unit_vector(const double *P, double Pu[3])
{
    static const double ez[3] = {0, 0, 1};
    if (!P) P = ez;
    double n = sqrt(P[0] * P[0] + P[1] * P[1] + P[2] * P[2]);
    if (!(n > 0)) return NMSO_E_ARG;
    Pu[0] = P[0] / n; Pu[1] = P[1] / n; Pu[2] = P[2] / n;
    return NMSO_OK;
}

/* amp: [8][nq] raw sums; out: [nk][nq]; also optionally the H-J vector Q: [6][nq] (Re/Im of Qx,Qy,Qz of the UNSCALED M~) */
int nmso_response(const double *amp, const double *theta, int64_t nq, const double *P,
                  double sN, double sM, double invV, const int *kinds, int nk, double *out, double *out_Q)
{
    double Pu[3];
    if (!amp || !theta || nq <= 0 || nk < 0 || (nk > 0 && (!kinds || !out))) return NMSO_E_ARG;
    if (unit_vector(P, Pu)) return NMSO_E_ARG;
    for (int a = 0; a < nk; ++a) if (kinds[a] < 0 || kinds[a] >= K_COUNT) return NMSO_E_ARG;
#pragma omp parallel for
    for (int64_t i = 0; i < nq; ++i) {
        const double complex An = sN * (amp[0 * nq + i] + I * amp[1 * nq + i]);
        const double complex M[3] = {sM * (amp[2 * nq + i] + I * amp[3 * nq + i]),
                                     sM * (amp[4 * nq + i] + I * amp[5 * nq + i]),
                                     sM * (amp[6 * nq + i] + I * amp[7 * nq + i])};
        double val[K_COUNT];
        responses_at_point(An, M, theta[i], Pu, invV, val);
        for (int a = 0; a < nk; ++a) out[(int64_t)a * nq + i] = val[kinds[a]];
        if (out_Q) {
            const double complex Mu[3] = {amp[2 * nq + i] + I * amp[3 * nq + i], amp[4 * nq + i] + I * amp[5 * nq + i],
                                          amp[6 * nq + i] + I * amp[7 * nq + i]};
            const double complex qh[3] = {0.0, sin(theta[i]), cos(theta[i])};
            double complex t[3], Q[3];
            cross3(qh, Mu, t);
            cross3(qh, t, Q);
            for (int a = 0; a < 3; ++a) { out_Q[(2 * a) * nq + i] = creal(Q[a]); out_Q[(2 * a + 1) * nq + i] = cimag(Q[a]); }
        }
    }
    return NMSO_OK;
}

/* ------------------------------------------------------------------------
 * Form factor / interparticle interference split, Eq. 49-50 (L376-L387),
 * extended to every kind B(A,A) (reading 13):
 *   total = B(sum_p A_p, sum_p A_p),   form = sum_p B(A_p, A_p),
 * A_p = amplitudes of particle p alone INCLUDING its centre r^p.
 * Loop over particles; each particle is a plain call of nmso_amplitudes.
 * ---------------------------------------------------------------------- */
int nmso_form_factor_split(const float *pos, const float *N, const float *m, int64_t W,
                           const int64_t *offsets, int64_t K, const float *centres, const double *R,
                           const double *qy, const double *qz, const double *theta, int64_t nq,
                           const double *P, double sN, double sM, double invV,
                           const int *kinds, int nk, double *out_total, double *out_form)
{
    if (!offsets || K <= 0 || offsets[0] != 0 || offsets[K] != W || nk <= 0) return NMSO_E_ARG;
    double *Ap = (double *)malloc(sizeof(double) * 8 * (size_t)nq);
    double *At = (double *)calloc(8 * (size_t)nq, sizeof(double));
    double *Bp = (double *)malloc(sizeof(double) * (size_t)nk * (size_t)nq);
    if (!Ap || !At || !Bp) { free(Ap); free(At); free(Bp); return NMSO_E_NOMEM; }
    memset(out_form, 0, sizeof(double) * (size_t)nk * (size_t)nq);
    int rc = NMSO_OK;
    for (int64_t p = 0; p < K && !rc; ++p) {
        const int64_t b = offsets[p], e = offsets[p + 1];
        if (e <= b) { if (e < b) rc = NMSO_E_ARG; continue; }
        const int64_t one[2] = {0, e - b};
        rc = nmso_amplitudes(pos + 3 * b, N ? N + b : NULL, m ? m + 3 * b : NULL, e - b,
                             centres ? one : NULL, centres ? 1 : 0, centres ? centres + 3 * p : NULL, R,
                             NULL, qy, qz, nq, Ap, NULL);
        if (rc) break;
        rc = nmso_response(Ap, theta, nq, P, sN, sM, invV, kinds, nk, Bp, NULL);
        if (rc) break;
        for (int64_t i = 0; i < (int64_t)nk * nq; ++i) out_form[i] += Bp[i];
        for (int64_t i = 0; i < 8 * nq; ++i) At[i] += Ap[i];
    }
    if (!rc) rc = nmso_response(At, theta, nq, P, sN, sM, invV, kinds, nk, out_total, NULL);
    free(Ap); free(At); free(Bp);
    return rc;
}

/* ------------------------------------------------------------------------
 * Angular modal decomposition, Eq. 31-33 (L187-L199).  On a polar grid with
 * theta_j = 2 pi j / n_theta (reading 7) the trapezoidal rule of Eq. 31
 * is the plain sum
 *   I_k^{s,c}(q_i) = (2 - delta_k0) / n_theta * sum_j f(q_i, theta_j) {sin, cos}(k theta_j),
 * with theta_j the grid's own (float32, promoted) angles.  Eq. 32: a_k = sum_i I_k(q_i).
 * Eq. 33: A_k = a_k / sum_{j=0..kmax} sqrt(a_j^s^2 + a_j^c^2) (0 where that sum is 0).
 * maps [nm][n0][n1]; Is, Ic [nm][kmax+1][n0]; as_, ac, As, Ac [nm][kmax+1].
 * ---------------------------------------------------------------------- */
int nmso_modal(const double *maps, int nm, int n0, int n1, const double *theta, int kmax,
               double *Is, double *Ic, double *as_, double *ac, double *As, double *Ac)
{
    if (!maps || !theta || !Is || !Ic || !as_ || !ac || !As || !Ac || nm <= 0 || n0 <= 0 || n1 <= 0 || kmax < 0)
        return NMSO_E_ARG;
    const int nk = kmax + 1;
    for (int a = 0; a < nm; ++a) {
        for (int k = 0; k < nk; ++k) {
            const double pref = (k == 0 ? 1.0 : 2.0) / (double)n1;
            double sa = 0.0, ca = 0.0;
            for (int i = 0; i < n0; ++i) {
                double ss = 0.0, cc = 0.0;
                for (int j = 0; j < n1; ++j) {
                    const double f = maps[((int64_t)a * n0 + i) * n1 + j];
                    ss += f * sin((double)k * theta[j]);
                    cc += f * cos((double)k * theta[j]);
                }
                Is[((int64_t)a * nk + k) * n0 + i] = pref * ss;
                Ic[((int64_t)a * nk + k) * n0 + i] = pref * cc;
                sa += pref * ss;
                ca += pref * cc;
            }
            as_[(int64_t)a * nk + k] = sa;
            ac[(int64_t)a * nk + k] = ca;
        }
        double norm = 0.0;
        for (int k = 0; k < nk; ++k)
            norm += sqrt(as_[(int64_t)a * nk + k] * as_[(int64_t)a * nk + k] + ac[(int64_t)a * nk + k] * ac[(int64_t)a * nk + k]);
        for (int k = 0; k < nk; ++k) {
            As[(int64_t)a * nk + k] = norm > 0.0 ? as_[(int64_t)a * nk + k] / norm : 0.0;
            Ac[(int64_t)a * nk + k] = norm > 0.0 ? ac[(int64_t)a * nk + k] / norm : 0.0;
        }
    }
    return NMSO_OK;
}

/* ------------------------------------------------------------------------
 * Azimuthal average, Eq. 30 (L181): I(q) = (1/2pi) int_0^2pi f(q,th) dth by the
 * trapezoidal rule (L183).  On the periodic grid th_j = 2 pi j / n_th, j < n_th,
 * the trapezoid is the arithmetic mean over j (reading 7).
 * maps: [nm][n0][n1] -> out [nm][n0].
 * ---------------------------------------------------------------------- */
int nmso_azimuthal_polar(const double *maps, int nm, int n0, int n1, double *out)
{
    if (!maps || !out || nm <= 0 || n0 <= 0 || n1 <= 0) return NMSO_E_ARG;
    for (int a = 0; a < nm; ++a)
        for (int i = 0; i < n0; ++i) {
            double s = 0.0;
            for (int j = 0; j < n1; ++j) s += maps[((int64_t)a * n0 + i) * n1 + j];
            out[(int64_t)a * n0 + i] = s / (double)n1;
        }
    return NMSO_OK;
}

/* Histogram average by |q| (reading 8; not in the paper, which only has polar grids L343):
 * bin = floor((|q| - q_lo) / (q_hi - q_lo) * n_bins) evaluated in fp64 exactly in this order,
 * |q| = sqrt(q_y^2 + q_z^2); points with |q| < q_lo or bin >= n_bins are dropped;
 * value = mean of members, empty bins give 0 with count 0. */
int nmso_azimuthal_hist(const double *maps, int nm, const double *qy, const double *qz, int64_t nq,
                        int n_bins, double q_lo, double q_hi, double *out_I, int32_t *out_count)
{
    if (!maps || !out_I || nm <= 0 || nq <= 0 || n_bins <= 0 || !(q_hi > q_lo)) return NMSO_E_ARG;
    int32_t *cnt = (int32_t *)calloc((size_t)n_bins, sizeof(int32_t));
    if (!cnt) return NMSO_E_NOMEM;
    memset(out_I, 0, sizeof(double) * (size_t)nm * (size_t)n_bins);
    for (int64_t i = 0; i < nq; ++i) {
        const double q = sqrt(qy[i] * qy[i] + qz[i] * qz[i]);
        if (q < q_lo) continue;
        const double fb = floor((q - q_lo) / (q_hi - q_lo) * (double)n_bins);
        if (!(fb < (double)n_bins)) continue;
        const int b = (int)fb;
        cnt[b] += 1;
        for (int a = 0; a < nm; ++a) out_I[(int64_t)a * n_bins + b] += maps[(int64_t)a * nq + i];
    }
    for (int a = 0; a < nm; ++a)
        for (int b = 0; b < n_bins; ++b)
            if (cnt[b] > 0) out_I[(int64_t)a * n_bins + b] /= (double)cnt[b];
    if (out_count) memcpy(out_count, cnt, sizeof(int32_t) * (size_t)n_bins);
    free(cnt);
    return NMSO_OK;
}

/* ------------------------------------------------------------------------
 * Two-dimensional correlation function, Eq. 36 (L213):
 *   C(rho, alpha) = int_0^2pi int_0^inf f(q, theta) exp(i q rho cos(theta - alpha)) q dq dtheta,
 * by the trapezoidal rule (L183) on the polar detector grid: periodic in theta (theta_j = 2 pi j / n1,
 * weight 2 pi / n1, reading 7), non-uniform in q over the available abscissae only, no
 * extrapolation to 0 or infinity (the reading taken for c(r), reading 9):
 *   wq_0 = (q_1 - q_0)/2, wq_i = (q_{i+1} - q_{i-1})/2, wq_{n0-1} = (q_{n0-1} - q_{n0-2})/2  (n0 = 1: wq = 1).
 * q cos(theta - alpha) rho = (q sin theta)(rho sin alpha) + (q cos theta)(rho cos alpha).
 * map [n0][n1]; q [n0], theta [n1], rho [m0], alpha [m1] (float32 grid values promoted); out_re, out_im [m0][m1].
 * ---------------------------------------------------------------------- */
int nmso_correlation_2d(const double *map, int n0, int n1, const double *q, const double *theta,
                        int m0, int m1, const double *rho, const double *alpha, double *out_re, double *out_im)
{
    if (!map || !q || !theta || !rho || !alpha || !out_re || !out_im || n0 <= 0 || n1 <= 0 || m0 <= 0 || m1 <= 0)
        return NMSO_E_ARG;
    const double dth = 2.0 * M_PI / (double)n1;
#pragma omp parallel for schedule(static)
    for (int64_t o = 0; o < (int64_t)m0 * m1; ++o) {
        const int a = (int)(o / m1), b = (int)(o % m1);
        const double ry = rho[a] * sin(alpha[b]), rz = rho[a] * cos(alpha[b]);
        double re = 0.0, im = 0.0;
        for (int i = 0; i < n0; ++i) {
            double wq = 1.0;
            if (n0 > 1) wq = i == 0 ? 0.5 * (q[1] - q[0]) : (i == n0 - 1 ? 0.5 * (q[n0 - 1] - q[n0 - 2]) : 0.5 * (q[i + 1] - q[i - 1]));
            for (int j = 0; j < n1; ++j) {
                const double w = map[(int64_t)i * n1 + j] * q[i] * wq * dth;
                const double ph = (q[i] * sin(theta[j])) * ry + (q[i] * cos(theta[j])) * rz;
                re += w * cos(ph);
                im += w * sin(ph);
            }
        }
        out_re[o] = re;
        out_im[o] = im;
    }
    return NMSO_OK;
}

/* ------------------------------------------------------------------------
 * Correlation function and pair-distance distribution, Eq. 34-35 (L205-L207):
 *   c(r) = (1/2pi^2) int I(q) j0(qr) q^2 dq,  p(r) = r^2 c(r),  j0(x) = sin x / x,
 * trapezoidal rule (L183) on the available abscissae, literally with the
 * 1/(2 pi^2) prefactor and without extrapolation to 0 or infinity
 * (reading 9).  Bins with count == 0 are skipped (count may be NULL).
 * I: [nm][nb], q: [nb] ascending; out_c, out_p: [nm][nr].
 * ---------------------------------------------------------------------- */
static double j0s(double x) { return fabs(x) < 1e-4 ? 1.0 - x * x / 6.0 : sin(x) / x; }

int nmso_correlation(const double *Iq, const double *q, const int32_t *count, int nm, int nb,
                     const double *r, int nr, double *out_c, double *out_p)
{
    if (!Iq || !q || !r || nm <= 0 || nb <= 0 || nr <= 0 || !out_c || !out_p) return NMSO_E_ARG;
    int *idx = (int *)malloc(sizeof(int) * (size_t)nb);
    if (!idx) return NMSO_E_NOMEM;
    int n = 0;
    for (int b = 0; b < nb; ++b) if (!count || count[b] > 0) idx[n++] = b;
#pragma omp parallel for
    for (int k = 0; k < nr; ++k)
        for (int a = 0; a < nm; ++a) {
            double s = 0.0;
            for (int t = 0; t + 1 < n; ++t) {
                const int b0 = idx[t], b1 = idx[t + 1];
                const double f0 = Iq[(int64_t)a * nb + b0] * j0s(q[b0] * r[k]) * q[b0] * q[b0];
                const double f1 = Iq[(int64_t)a * nb + b1] * j0s(q[b1] * r[k]) * q[b1] * q[b1];
                s += 0.5 * (f0 + f1) * (q[b1] - q[b0]);
            }
            const double c = s / (2.0 * M_PI * M_PI);
            out_c[(int64_t)a * nr + k] = c;
            out_p[(int64_t)a * nr + k] = r[k] * r[k] * c;
        }
    free(idx);
    return NMSO_OK;
}
