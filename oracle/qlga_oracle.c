/*
 * oracle/qlga_oracle.c  --  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded CPU implementation of the spin-2 BEC quantum
 * lattice gas algorithm (QLGA) time step of arXiv:1907.12834, written from the
 * paper one operator at a time, whole-lattice arrays, no fusion, no
 * stencil shortcut, no blocking.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, table or helper with the CUDA path under
 * paper_1907_12834_b200/csrc/.
 *
 * Real type: `REAL` (default double; build with -DREAL="long double" for the
 * extended-precision arbiter).  Complex = C99 `REAL _Complex`.
 *
 * State layout:  q[j][sigma][y][x]  complex,
 *   j = 0..4 <-> m_f = +2,+1,0,-1,-2 ; sigma = 0,1 <-> spinor component 1,2 ;
 *   x fastest; periodic in x (and y in 2D, z in 3D; ny = nz = 1 in 1D); 3D: q[j][sigma][z][y][x].
 *   Bosonic field psi_m = q_{m1} + q_{m2}.
 *
 * Readings of the paper where it is silent (R1..R9) are
 * marked [Rn] below.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): unitarity, Fourier symbol of the
 * kinetic factor incl. eq. (109), Table I eigenstates (tests/golden/table1.json),
 * scipy.linalg.expm of the dense 5x5 (and 10x10) interaction Hamiltonian,
 * bright/dark soliton stationarity, Galilean drift, exact covariances,
 * vorticity quantisation / winding.  No function here is "parity unpinned"
 * except the conventions listed as such in DESIGN.md (R6 split, R7 x-before-y).
 */
#include <complex.h>
#include <math.h>
#include <tgmath.h>
#include <stdlib.h>
#include <string.h>

#ifndef REAL
#define REAL double
#endif
typedef REAL real;
typedef REAL _Complex cplx;

#define NM 5            /* Zeeman levels m = +2..-2 */
#define NS 2            /* spinor components per level */

static inline long wrapl(long i, long n) { i %= n; return i < 0 ? i + n : i; }

size_t orc_sizeof_real(void) { return sizeof(real); }

/* q1 = q2 = psi/2  [R6]  (psi: [5][ny][nx], q: [5][2][ny][nx]) */
void orc_split_psi(const cplx *psi, cplx *q, long nx, long ny, long nz)
{
    long n = nx * ny * nz;
    for (int j = 0; j < NM; ++j)
        for (long r = 0; r < n; ++r) {
            cplx h = psi[(size_t)j * n + r] / (real)2;
            q[((size_t)j * NS + 0) * n + r] = h;
            q[((size_t)j * NS + 1) * n + r] = h;
        }
}

/* psi_m = q_m1 + q_m2 */
void orc_psi_of_q(const cplx *q, cplx *psi, long nx, long ny, long nz)
{
    long n = nx * ny * nz;
    for (int j = 0; j < NM; ++j)
        for (long r = 0; r < n; ++r)
            psi[(size_t)j * n + r] = q[((size_t)j * NS + 0) * n + r] + q[((size_t)j * NS + 1) * n + r];
}

/* ------------------------------------------------------------------------
 * Collide  [R1]  (operator "C" of eq. 107):
 *   (q1, q2) -> (a q1 + b q2, b q1 + a q2),  a = (1-i)/2, b = (1+i)/2
 * the square-root-of-swap matrix, at every site and for every m.
 * ---------------------------------------------------------------------- */
void orc_collide(cplx *q, long nx, long ny, long nz)
{
    const cplx a = ((real)1 - I) / (real)2;
    const cplx b = ((real)1 + I) / (real)2;
    long n = nx * ny * nz;
    for (int j = 0; j < NM; ++j)
        for (long r = 0; r < n; ++r) {
            cplx q1 = q[((size_t)j * NS + 0) * n + r];
            cplx q2 = q[((size_t)j * NS + 1) * n + r];
            q[((size_t)j * NS + 0) * n + r] = a * q1 + b * q2;
            q[((size_t)j * NS + 1) * n + r] = b * q1 + a * q2;
        }
}

/* ------------------------------------------------------------------------
 * Stream  [R2]  (operators S_i, S_i^T of eq. 107):
 *   transpose = 0 :  (S_{d,sigma} q)_sigma(r)   = q_sigma(r - e_d)
 *   transpose = 1 :  (S^T_{d,sigma} q)_sigma(r) = q_sigma(r + e_d)
 * for all five m at once, periodic; the other spinor component is untouched.
 * d = 0 (x) or 1 (y); sigma = 0,1 <-> component 1,2.
 * ---------------------------------------------------------------------- */
void orc_stream(cplx *q, long nx, long ny, long nz, int d, int sigma, int transpose)
{
    long n = nx * ny * nz;
    cplx *tmp = (cplx *)malloc(sizeof(cplx) * (size_t)n);
    long sh = transpose ? +1 : -1;          /* new(r) = old(r + sh e_d) */
    for (int j = 0; j < NM; ++j) {
        cplx *p = q + ((size_t)j * NS + (size_t)sigma) * n;
        memcpy(tmp, p, sizeof(cplx) * (size_t)n);
        for (long z = 0; z < nz; ++z)
            for (long y = 0; y < ny; ++y)
                for (long x = 0; x < nx; ++x) {
                    long xs = (d == 0) ? wrapl(x + sh, nx) : x;
                    long ys = (d == 1) ? wrapl(y + sh, ny) : y;
                    long zs = (d == 2) ? wrapl(z + sh, nz) : z;
                    p[(z * ny + y) * nx + x] = tmp[(zs * ny + ys) * nx + xs];
                }
    }
    free(tmp);
}

/* Kinetic factor  I'_{d,sigma} = S C S^T C   (eq. 107),
 * rightmost operator applied first. */
void orc_kinetic_factor(cplx *q, long nx, long ny, long nz, int d, int sigma)
{
    orc_collide(q, nx, ny, nz);
    orc_stream(q, nx, ny, nz, d, sigma, 1);
    orc_collide(q, nx, ny, nz);
    orc_stream(q, nx, ny, nz, d, sigma, 0);
}

/* ------------------------------------------------------------------------
 * Spin-2 matrices  [R5b]  (eq. 36 is missing from the text, PAPER.md:265-267;
 * "their usual spin-2 SU(2) representations"):
 *   (f_z)_{mm} = m,   f_+ |m> = sqrt(6 - m(m+1)) |m+1>,   f_- = f_+^T,
 *   f_x = (f_+ + f_-)/2,   f_y = (f_+ - f_-)/(2i),   index j = 2 - m.
 * ---------------------------------------------------------------------- */
static cplx FX[NM][NM], FY[NM][NM], FZ[NM][NM];
static int spin_ready = 0;

static void build_spin_matrices(void)
{
    real fp[NM][NM];
    memset(fp, 0, sizeof fp);
    memset(FX, 0, sizeof FX); memset(FY, 0, sizeof FY); memset(FZ, 0, sizeof FZ);
    for (int j = 1; j < NM; ++j) {               /* |m> with m = 2-j  ->  |m+1> = row j-1 */
        int m = 2 - j;
        fp[j - 1][j] = sqrt((real)(6 - m * (m + 1)));
    }
    for (int r = 0; r < NM; ++r)
        for (int c = 0; c < NM; ++c) {
            real plus = fp[r][c], minus = fp[c][r];
            FX[r][c] = (plus + minus) / (real)2;
            FY[r][c] = (plus - minus) / ((real)2 * I);
        }
    for (int j = 0; j < NM; ++j) FZ[j][j] = (real)(2 - j);
    spin_ready = 1;
}

/* copy the spin matrices out (tests check the su(2) algebra on them) */
void orc_spin_matrices(cplx *fx, cplx *fy, cplx *fz)
{
    if (!spin_ready) build_spin_matrices();
    memcpy(fx, FX, sizeof FX); memcpy(fy, FY, sizeof FY); memcpy(fz, FZ, sizeof FZ);
}

/* Local mean-field quantities at one site, from psi[5]:
 *   rho = sum_m |psi_m|^2                                    eq. (3), (38a)
 *   F_nu = sum_{mm'} (f_nu)_{mm'} psi_m^* psi_m'             eq. (5)
 *   chi_m = (-1)^m psi_{-m}^*      (time-reversed spinor)     [R5]
 *   Theta = <chi|psi> = 2 psi_2 psi_-2 - 2 psi_1 psi_-1 + psi_0^2 = sqrt(5) A00   eq. (4), (35)
 */
static void site_fields(const cplx psi[NM], real *rho, real F[3], cplx chi[NM], cplx *theta)
{
    if (!spin_ready) build_spin_matrices();
    real r = 0;
    cplx fx = 0, fy = 0, fz = 0, th = 0;
    for (int a = 0; a < NM; ++a) {
        r += creal(psi[a]) * creal(psi[a]) + cimag(psi[a]) * cimag(psi[a]);
        for (int b = 0; b < NM; ++b) {
            cplx pp = conj(psi[a]) * psi[b];
            fx += FX[a][b] * pp; fy += FY[a][b] * pp; fz += FZ[a][b] * pp;
        }
    }
    for (int j = 0; j < NM; ++j) {
        real sgn = (j % 2 == 0) ? (real)1 : (real)-1;      /* (-1)^m = (-1)^j, m = 2-j */
        chi[j] = sgn * conj(psi[NM - 1 - j]);
    }
    for (int j = 0; j < NM; ++j) th += conj(chi[j]) * psi[j];
    *rho = r; F[0] = creal(fx); F[1] = creal(fy); F[2] = creal(fz); *theta = th;
}

/* Dense 5x5 interaction Hamiltonian without the scalar part  [R4][R5]:
 *   K = c1 (F_x f_x + F_y f_y + F_z f_z) + (c2/5) |chi><chi|
 * so that H_int[psi] = c0 rho 1 + K, i.e. the right-hand side of eq. (34),
 * PAPER.md:258, with its coefficients frozen at the current psi. */
static void site_K(const cplx psi[NM], real c1, real c2, cplx K[NM][NM], real *rho)
{
    real F[3]; cplx chi[NM], th;
    site_fields(psi, rho, F, chi, &th);
    for (int a = 0; a < NM; ++a)
        for (int b = 0; b < NM; ++b)
            K[a][b] = c1 * (F[0] * FX[a][b] + F[1] * FY[a][b] + F[2] * FZ[a][b])
                    + (c2 / (real)5) * chi[a] * conj(chi[b]);
}

/* export H_int = c0 rho + K for one site (tests compare exp(-i s H) with scipy) */
void orc_site_hamiltonian(const cplx *psi, real c0, real c1, real c2, cplx *H)
{
    cplx K[NM][NM]; real rho;
    site_K(psi, c1, c2, K, &rho);
    for (int a = 0; a < NM; ++a)
        for (int b = 0; b < NM; ++b)
            H[a * NM + b] = K[a][b] + ((a == b) ? c0 * rho : (real)0);
}

/* v <- exp(-i s K) v  by the Taylor polynomial of the exponential applied to the
 * vector in Horner form,
 *     u_p = v,   u_{k-1} = v + (-i s / k) K u_k   (k = p..1),   result u_0,
 * with the degree p chosen from the bound theta = |s| max_a sum_b |K_ab| >= |s| ||K||
 * so that the first dropped term theta^(p+1)/(p+1)! is below 1e-30 (far below one
 * ulp of either real type); angles above 1/2 are split into equal sub-angles.  Horner form matters: adding the terms one after the
 * other to the running sum silently drops the small same-signed even-order terms
 * (a term below half an ulp of a representable sum is always rounded away), a
 * systematic norm loss of ~1e-17 per application that breaks the 1e-13/1000-step
 * unitarity pin; in Horner form the small terms meet first and the one rounding
 * of the final addition is unbiased. */
static void expm_apply(cplx K[NM][NM], real s, cplx v[NM])
{
    real theta = 0;
    for (int a = 0; a < NM; ++a) {
        real row = 0;
        for (int b = 0; b < NM; ++b) row += fabs(creal(K[a][b])) + fabs(cimag(K[a][b]));
        if (row > theta) theta = row;
    }
    theta *= fabs(s);
    /* large angles: exp(-i s K) = [exp(-i (s/n) K)]^n exactly (K is fixed), with n
     * chosen so that each factor has theta/n <= 1/2 and the alternating series
     * suffers no cancellation */
    int nsub = 1;
    if (theta > (real)0.5) nsub = (int)ceil(theta / (real)0.5);
    real ss = s / (real)nsub, th = theta / (real)nsub;
    int p = 1;
    real bound = th * th / (real)2;                 /* th^(p+1)/(p+1)! for p = 1 */
    while (bound > (real)1e-30 && p < 200) { ++p; bound *= th / (real)(p + 1); }

    cplx u[NM], w[NM], v0[NM];
    for (int a = 0; a < NM; ++a) u[a] = v[a];
    for (int rep = 0; rep < nsub; ++rep) {
        for (int a = 0; a < NM; ++a) v0[a] = u[a];
        for (int k = p; k >= 1; --k) {
            for (int a = 0; a < NM; ++a) {
                cplx acc = 0;
                for (int b = 0; b < NM; ++b) acc += K[a][b] * u[b];
                w[a] = acc;
            }
            for (int a = 0; a < NM; ++a) u[a] = v0[a] + (-I * ss / (real)k) * w[a];
        }
    }
    for (int a = 0; a < NM; ++a) v[a] = u[a];
}

/* ------------------------------------------------------------------------
 * Interaction  U^{(s)}  [R4]  (operator "U" of eq. 108 / "U^{1/4}" of eq. 112,
 * PAPER.md:1036-1053): at every site, from the current state,
 *   W = exp(-i s H_int[psi]),   q_{.,sigma} <- W q_{.,sigma}  for sigma = 1, 2,
 * evaluated as  exp(-i s c0 rho) * exp(-i s K)  (the scalar part commutes).
 * ---------------------------------------------------------------------- */
/* With a chemical potential (section II.C: "a chemical potential term of the
 * form mu psi_m"; eq. (75), E = mu + p^2 - k^2): H_int + mu 1, i.e. one more scalar
 * phase exp(-i s mu).  mu = 0 is the paper's own simulations (bit-identical to the form without). */
void orc_interaction_mu(cplx *q, long nx, long ny, long nz, real c0, real c1, real c2, real mu, real s)
{
    long n = nx * ny * nz;
    for (long r = 0; r < n; ++r) {
        cplx psi[NM], K[NM][NM], v[NM];
        real rho;
        for (int j = 0; j < NM; ++j)
            psi[j] = q[((size_t)j * NS + 0) * n + r] + q[((size_t)j * NS + 1) * n + r];
        site_K(psi, c1, c2, K, &rho);
        cplx phase = exp(-I * (s * c0 * rho + s * mu));
        for (int sg = 0; sg < NS; ++sg) {
            for (int j = 0; j < NM; ++j) v[j] = q[((size_t)j * NS + sg) * n + r];
            expm_apply(K, s, v);
            for (int j = 0; j < NM; ++j) q[((size_t)j * NS + sg) * n + r] = phase * v[j];
        }
    }
}

void orc_interaction(cplx *q, long nx, long ny, long nz, real c0, real c1, real c2, real s)
{
    orc_interaction_mu(q, nx, ny, nz, c0, c1, c2, (real)0, s);
}

/* ------------------------------------------------------------------------
 * One time step  (rightmost operator first):
 *   order 0, plain       eq. (108):  I'_{x1} I'_{x1} I'_{x2} I'_{x2} U
 *   order 1, interleaved eq. (112):  I'_{x1}U^{1/4} I'_{x1}U^{1/4} I'_{x2}U^{1/4} I'_{x2}U^{1/4}
 *   2D  [R7] ("n = 8"): the four y factors act before the four
 *   x factors, U (plain) or U^{1/8} (interleaved, before every factor).
 *   3D  ("n = 12"): z factors, then y, then x; U^{1/12}.
 * ---------------------------------------------------------------------- */
void orc_step_mu(cplx *q, long nx, long ny, long nz, int ndim, real c0, real c1, real c2, real mu,
                 int order, long nsteps)
{
    const int nfac = 4 * ndim;
    for (long t = 0; t < nsteps; ++t) {
        if (order == 0) orc_interaction_mu(q, nx, ny, nz, c0, c1, c2, mu, (real)1);
        for (int d = ndim - 1; d >= 0; --d)              /* y factors first, then x */
            for (int k = 0; k < 4; ++k) {
                int sigma = (k < 2) ? 1 : 0;             /* component 2, 2, 1, 1 */
                if (order == 1) orc_interaction_mu(q, nx, ny, nz, c0, c1, c2, mu, (real)1 / (real)nfac);
                orc_kinetic_factor(q, nx, ny, nz, d, sigma);
            }
    }
}

void orc_step(cplx *q, long nx, long ny, long nz, int ndim, real c0, real c1, real c2,
              int order, long nsteps)
{
    orc_step_mu(q, nx, ny, nz, ndim, c0, c1, c2, (real)0, order, nsteps);
}

/* ------------------------------------------------------------------------
 * Observables (sums over the lattice; out[] is always double):
 *   out[0..4]  n_m      = sum_r |psi_m|^2                        eq. (3)
 *   out[5]     norm_psi = sum_m n_m
 *   out[6]     norm_q   = sum_{r,m,sigma} |q|^2   (the unitary invariant)
 *   out[7..9]  F_x,F_y,F_z = sum_r <psi|f_nu|psi>                eq. (5), (59)-(60)
 *   out[10,11] A00 = sum_r A00(r),  A00(r) = Theta(r)/sqrt(5)    eq. (4), (35) [R5c]
 *   out[12]    sum_r |A00(r)|^2
 *   out[13]    e_kin = sum_r sum_m sum_d |psi_m(r+e_d) - psi_m(r)|^2    (eq. 12, hbar=1, m=1/2)
 *   out[14]    e_c0  = (c0/2) sum rho^2                          eq. (32)
 *   out[15]    e_c1  = (c1/2) sum |F|^2
 *   out[16]    e_c2  = (c2/2) sum |A00|^2
 *   out[17]    e_total = e_kin + e_c0 + e_c1 + e_c2              [R9]
 *   out[18,19] e_dt = i(<psi|psi> - <psi|psi_prev>)/<psi|psi>    eq. (85)
 *              (NaN if qprev == NULL), <a|b> = sum_{r,m} a_m^* b_m.
 * ---------------------------------------------------------------------- */
void orc_observables(const cplx *q, const cplx *qprev, long nx, long ny, long nz, int ndim,
                     real c0, real c1, real c2, double *out)
{
    long n = nx * ny * nz;
    real nm[NM] = {0, 0, 0, 0, 0}, normq = 0, Fs[3] = {0, 0, 0}, a2 = 0;
    real ekin = 0, s_rho2 = 0, s_F2 = 0;
    cplx a00 = 0, ov = 0;
    const real rt5 = sqrt((real)5);
    for (long zz = 0; zz < nz; ++zz)
    for (long y = 0; y < ny; ++y)
        for (long x = 0; x < nx; ++x) {
            long r = (zz * ny + y) * nx + x;
            cplx psi[NM], chi[NM], th;
            real rho, F[3];
            for (int j = 0; j < NM; ++j) {
                cplx q1 = q[((size_t)j * NS + 0) * n + r], q2 = q[((size_t)j * NS + 1) * n + r];
                psi[j] = q1 + q2;
                normq += creal(q1) * creal(q1) + cimag(q1) * cimag(q1)
                       + creal(q2) * creal(q2) + cimag(q2) * cimag(q2);
                nm[j] += creal(psi[j]) * creal(psi[j]) + cimag(psi[j]) * cimag(psi[j]);
            }
            site_fields(psi, &rho, F, chi, &th);
            for (int k = 0; k < 3; ++k) Fs[k] += F[k];
            cplx A = th / rt5;
            a00 += A;
            a2 += creal(A) * creal(A) + cimag(A) * cimag(A);
            s_rho2 += rho * rho;
            s_F2 += F[0] * F[0] + F[1] * F[1] + F[2] * F[2];
            for (int d = 0; d < ndim; ++d) {
                long xn = (d == 0) ? wrapl(x + 1, nx) : x;
                long yn = (d == 1) ? wrapl(y + 1, ny) : y;
                long zn = (d == 2) ? wrapl(zz + 1, nz) : zz;
                long rn = (zn * ny + yn) * nx + xn;
                for (int j = 0; j < NM; ++j) {
                    cplx pn = q[((size_t)j * NS + 0) * n + rn] + q[((size_t)j * NS + 1) * n + rn];
                    cplx df = pn - psi[j];
                    ekin += creal(df) * creal(df) + cimag(df) * cimag(df);
                }
            }
            if (qprev)
                for (int j = 0; j < NM; ++j) {
                    cplx pp = qprev[((size_t)j * NS + 0) * n + r] + qprev[((size_t)j * NS + 1) * n + r];
                    ov += conj(psi[j]) * pp;
                }
        }
    real npsi = 0;
    for (int j = 0; j < NM; ++j) { out[j] = (double)nm[j]; npsi += nm[j]; }
    out[5] = (double)npsi; out[6] = (double)normq;
    out[7] = (double)Fs[0]; out[8] = (double)Fs[1]; out[9] = (double)Fs[2];
    out[10] = (double)creal(a00); out[11] = (double)cimag(a00); out[12] = (double)a2;
    real e0 = c0 / (real)2 * s_rho2, e1 = c1 / (real)2 * s_F2, e2 = c2 / (real)2 * a2;
    out[13] = (double)ekin; out[14] = (double)e0; out[15] = (double)e1; out[16] = (double)e2;
    out[17] = (double)(ekin + e0 + e1 + e2);
    if (qprev) {
        cplx e = I * (npsi - ov) / npsi;
        out[18] = (double)creal(e); out[19] = (double)cimag(e);
    } else {
        out[18] = NAN; out[19] = NAN;
    }
}

/* ------------------------------------------------------------------------
 * Lattice vorticity, 2D  [R8]  (eq. 99-104).  Per m:
 *   v_x(r) = (1/2) arg( psi(r+e_x) psi^*(r-e_x) )     eq. (104a), phase difference wrapped
 *   v_y(r) = (1/2) arg( psi(r+e_y) psi^*(r-e_y) )     eq. (104b)
 *   omega(r) = (1/2)[ v_y(r+e_x) - v_y(r-e_x) - v_x(r+e_y) + v_x(r-e_y) ]
 * the symmetric-difference (eq. 102) curl of eq. (99); arg(0) := 0.
 * omega: [5][ny][nx] real.
 * ---------------------------------------------------------------------- */
static real arg0(cplx z)
{
    if (creal(z) == 0 && cimag(z) == 0) return 0;
    return atan2(cimag(z), creal(z));
}

void orc_vorticity(const cplx *q, long nx, long ny, real *omega)
{
    long n = nx * ny;
    cplx *psi = (cplx *)malloc(sizeof(cplx) * (size_t)n);
    real *vx = (real *)malloc(sizeof(real) * (size_t)n);
    real *vy = (real *)malloc(sizeof(real) * (size_t)n);
    for (int j = 0; j < NM; ++j) {
        for (long r = 0; r < n; ++r)
            psi[r] = q[((size_t)j * NS + 0) * n + r] + q[((size_t)j * NS + 1) * n + r];
        for (long y = 0; y < ny; ++y)
            for (long x = 0; x < nx; ++x) {
                long xp = wrapl(x + 1, nx), xm = wrapl(x - 1, nx);
                long yp = wrapl(y + 1, ny), ym = wrapl(y - 1, ny);
                vx[y * nx + x] = arg0(psi[y * nx + xp] * conj(psi[y * nx + xm])) / (real)2;
                vy[y * nx + x] = arg0(psi[yp * nx + x] * conj(psi[ym * nx + x])) / (real)2;
            }
        for (long y = 0; y < ny; ++y)
            for (long x = 0; x < nx; ++x) {
                long xp = wrapl(x + 1, nx), xm = wrapl(x - 1, nx);
                long yp = wrapl(y + 1, ny), ym = wrapl(y - 1, ny);
                omega[(size_t)j * n + y * nx + x] =
                    (vy[y * nx + xp] - vy[y * nx + xm] - vx[yp * nx + x] + vx[ym * nx + x]) / (real)2;
            }
    }
    free(psi); free(vx); free(vy);
}

/* ------------------------------------------------------------------------
 * Total density and the L2 error of eq. (115), PAPER.md:1074:
 *   rho(r) = sum_m |psi_m(r)|^2 = psi psi^dagger,
 *   epsilon = sum_lattice ( rho_ref(r) - rho(r) )^2 .
 * (the convergence study of Figs. 23-24.)
 * ---------------------------------------------------------------------- */
void orc_density(const cplx *q, long nx, long ny, long nz, real *rho)
{
    long n = nx * ny * nz;
    for (long r = 0; r < n; ++r) {
        real s = 0;
        for (int j = 0; j < NM; ++j) {
            cplx p = q[((size_t)j * NS + 0) * n + r] + q[((size_t)j * NS + 1) * n + r];
            s += creal(p) * creal(p) + cimag(p) * cimag(p);
        }
        rho[r] = s;
    }
}

double orc_density_l2_error(const cplx *q, const real *rho_ref, long nx, long ny, long nz)
{
    long n = nx * ny * nz;
    real *rho = (real *)malloc(sizeof(real) * (size_t)n);
    orc_density(q, nx, ny, nz, rho);
    real e = 0;
    for (long r = 0; r < n; ++r) { real d = rho_ref[r] - rho[r]; e += d * d; }
    free(rho);
    return (double)e;
}

/* ------------------------------------------------------------------------
 * Plaquette winding numbers (vortex detection; the
 * paper tracks "vortices with a positive / negative winding number", Figs. 18, 21,
 * 22, without printing the detector)  [R15]:
 * for the elementary plaquette with lower-left corner (x, y), corners taken
 * counter-clockwise  a=(x,y), b=(x+1,y), c=(x+1,y+1), d=(x,y+1),
 *   w(x,y) = [ arg(b a*) + arg(c b*) + arg(d c*) + arg(a d*) ] / (2 pi)  in {-1, 0, +1},
 * every phase difference wrapped to (-pi, pi] by taking arg of the product and
 * arg(0) := 0, rounded to the nearest integer.  wind: [5][ny][nx] int32.
 * ---------------------------------------------------------------------- */
void orc_winding(const cplx *q, long nx, long ny, int *wind)
{
    long n = nx * ny;
    const real twopi = (real)6.283185307179586476925286766559005768L;
    for (int j = 0; j < NM; ++j)
        for (long y = 0; y < ny; ++y)
            for (long x = 0; x < nx; ++x) {
                long xp = wrapl(x + 1, nx), yp = wrapl(y + 1, ny);
                long ia = y * nx + x, ib = y * nx + xp, ic = yp * nx + xp, id = yp * nx + x;
                cplx a = q[((size_t)j * NS + 0) * n + ia] + q[((size_t)j * NS + 1) * n + ia];
                cplx b = q[((size_t)j * NS + 0) * n + ib] + q[((size_t)j * NS + 1) * n + ib];
                cplx c = q[((size_t)j * NS + 0) * n + ic] + q[((size_t)j * NS + 1) * n + ic];
                cplx d = q[((size_t)j * NS + 0) * n + id] + q[((size_t)j * NS + 1) * n + id];
                real circ = arg0(b * conj(a)) + arg0(c * conj(b)) + arg0(d * conj(c)) + arg0(a * conj(d));
                wind[(size_t)j * n + ia] = (int)lrint((double)(circ / twopi));
            }
}

/* ------------------------------------------------------------------------
 * Association of two vortex detections (vortex tracking; the paper follows
 * "vortices with a positive / negative winding number" as red / blue tracks, Figs. 18, 21, 22,
 * PAPER.md:971-999, and does not print its tracker)  [R18]:
 * records (j, x, y, w) as rows of int[4] (the non-zero entries of orc_winding).  Two records can be the
 * same vortex at two times only if they agree in channel j and winding w.  d2 = periodic (minimal-image)
 * squared lattice distance.  The nearest candidate of a record is the record of the other list with the
 * same (j, w) and d2 <= max_d2 that comes first in the order (d2, y, x); two records are matched iff each
 * is the other's nearest candidate.  match_cur[i] = index into prev or -1, match_prev[k] = index into cur or -1.
 * Written as the definition: all pairs, no spatial search structure.
 * Pins (tests/test_oracle_tracking.py): hand-made cases (wrap-around distance, sign and channel mismatch,
 * the cut-off, a tie, a non-mutual pair), invariance under permutation of the lists, and the tracked speed
 * 2p of a kicked Pade quadrupole (eq. 71 with the units pinned by PAPER.md:906, 922).
 * ---------------------------------------------------------------------- */
static long match_d2(const int *a, const int *b, long nx, long ny)
{
    long dx = labs((long)a[1] - (long)b[1]), dy = labs((long)a[2] - (long)b[2]);
    if (nx - dx < dx) dx = nx - dx;
    if (ny - dy < dy) dy = ny - dy;
    return dx * dx + dy * dy;
}

static void nearest_candidates(const int *a, long na, const int *b, long nb, long nx, long ny, long max_d2, int *nn)
{
    for (long i = 0; i < na; ++i) {
        long best = -1, best_d2 = 0;
        for (long k = 0; k < nb; ++k) {
            if (b[4 * k] != a[4 * i] || b[4 * k + 3] != a[4 * i + 3]) continue;
            long d2 = match_d2(a + 4 * i, b + 4 * k, nx, ny);
            if (d2 > max_d2) continue;
            int first = best < 0 || d2 < best_d2
                     || (d2 == best_d2 && (b[4 * k + 2] < b[4 * best + 2]
                                           || (b[4 * k + 2] == b[4 * best + 2] && b[4 * k + 1] < b[4 * best + 1])));
            if (first) { best = k; best_d2 = d2; }
        }
        nn[i] = (int)best;
    }
}

void orc_vortex_match(const int *prev, long np, const int *cur, long nc, long nx, long ny, long max_d2,
                      int *match_cur, int *match_prev)
{
    int *nn_cur = (int *)malloc(sizeof(int) * (size_t)(nc > 0 ? nc : 1));
    int *nn_prev = (int *)malloc(sizeof(int) * (size_t)(np > 0 ? np : 1));
    nearest_candidates(cur, nc, prev, np, nx, ny, max_d2, nn_cur);
    nearest_candidates(prev, np, cur, nc, nx, ny, max_d2, nn_prev);
    for (long i = 0; i < nc; ++i) match_cur[i] = (nn_cur[i] >= 0 && nn_prev[nn_cur[i]] == i) ? nn_cur[i] : -1;
    for (long k = 0; k < np; ++k) match_prev[k] = (nn_prev[k] >= 0 && nn_cur[nn_prev[k]] == k) ? nn_prev[k] : -1;
    free(nn_cur); free(nn_prev);
}
