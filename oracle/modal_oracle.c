/*
 * modal_oracle.c -- ORACLE (test infrastructure, NOT the product).
 *
 * Plain, slow, fp64 CPU restatement of the modal equations of arXiv 2505.05940
 * (section 2 "Background"): sine modal bases, modal oscillator
 * coefficients (Eq. 13-14), von Karman coupling coefficients (Eq. 10-11), the
 * tension-modulation force (Eq. 8), the von Karman force (Eq. 9), the
 * Stormer-Verlet (Eq. 20-23) and FTM / impulse-invariant (Eq. 16-19) two-step
 * schemes, the stepping loop and the discrete energy of the lossless scheme.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may build, load or call this file.  It shares no code, header,
 * table or helper with paper_2505_05940_b200/ (the CUDA path) and is written in
 * the paper's order and notation: no blocking, no fusion, no reordering beyond
 * what each cited passage states.  OpenMP is used over independent batch
 * samples only; every inner loop is the plain definition.
 *
 * Readings of garbled / silent passages are listed in DESIGN.md ("Readings"),
 * ids R1..R14, and cited inline.
 *
 * Pins (tests/test_oracle_*.py): see the table in DESIGN.md.  No function in
 * this file is "parity unpinned"; the *harness constants* (loss parameters,
 * string pluck width, EA closure) have no source in the paper and are listed
 * as such in DESIGN.md.
 */
#include <math.h>
#include <stddef.h>
#include <stdlib.h>
#include <string.h>

#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_PI 3.14159265358979323846264338327950288

/* ------------------------------------------------------------------------ */
/* 1. Modal bases (Eq. 2: Laplacian eigenpairs).             */
/* ------------------------------------------------------------------------ */

/* Fixed string: Phi_m(x) = sqrt(2/L) sin(m pi x / L), lambda_m = (m pi/L)^2.
 * Unit L2 norm (reading R6).  m = 1..N. */
void orc_string_lambda(double L, int N, double *lambda)
{
    for (int m = 1; m <= N; ++m) {
        double a = m * ORC_PI / L;
        lambda[m - 1] = a * a;
    }
}

double orc_string_mode(int m, double L, double x)
{
    return sqrt(2.0 / L) * sin(m * ORC_PI * x / L);
}

/* Simply supported rectangle: Phi_{m,n}(x,y) = 2/sqrt(Lx Ly) sin(m pi x/Lx)
 * sin(n pi y/Ly), lambda = (m pi/Lx)^2 + (n pi/Ly)^2.  Returns the N smallest
 * lambda over the lattice m,n >= 1, ascending, ties broken by (m, then n)
 * (SPEC.md:117).  Plain exhaustive enumeration over an M x M lattice with M
 * large enough that every lattice point outside it has a larger lambda than
 * the N-th kept one; then an insertion sort.  Returns 0 on success. */
int orc_rect_modes(double Lx, double Ly, int N, int *m_out, int *n_out, double *lambda_out)
{
    /* The N points (1..N,1) all have lambda <= lmaxx and the N points (1,1..N) all have
     * lambda <= lmaxy, so the N-th smallest lambda is <= bound = min(lmaxx, lmaxy).
     * Every point with m > M or n > M is above the bound once ((M+1) pi/L)^2 > bound on
     * both axes, so an M x M lattice then holds all N smallest. */
    int M = N + 2;
    double lmaxx = (N * ORC_PI / Lx) * (N * ORC_PI / Lx) + (ORC_PI / Ly) * (ORC_PI / Ly);
    double lmaxy = (ORC_PI / Lx) * (ORC_PI / Lx) + (N * ORC_PI / Ly) * (N * ORC_PI / Ly);
    double bound = lmaxx < lmaxy ? lmaxx : lmaxy; /* N points lie at or below this */
    /* grow M until the first excluded row and column are above the bound */
    for (;;) {
        double lx = ((M + 1) * ORC_PI / Lx) * ((M + 1) * ORC_PI / Lx);
        double ly = ((M + 1) * ORC_PI / Ly) * ((M + 1) * ORC_PI / Ly);
        if (lx > bound && ly > bound) break;
        M *= 2;
    }
    size_t cnt = (size_t)M * (size_t)M;
    int *mm = (int *)malloc(cnt * sizeof(int));
    int *nn = (int *)malloc(cnt * sizeof(int));
    double *ll = (double *)malloc(cnt * sizeof(double));
    if (!mm || !nn || !ll) { free(mm); free(nn); free(ll); return 1; }
    size_t c = 0;
    for (int m = 1; m <= M; ++m)
        for (int n = 1; n <= M; ++n) {
            double a = m * ORC_PI / Lx, b = n * ORC_PI / Ly;
            mm[c] = m; nn[c] = n; ll[c] = a * a + b * b; ++c;
        }
    /* selection of the N smallest by repeated minimum (obviously correct) */
    for (int k = 0; k < N; ++k) {
        size_t best = (size_t)-1;
        for (size_t i = 0; i < cnt; ++i) {
            if (mm[i] == 0) continue; /* already taken */
            if (best == (size_t)-1) { best = i; continue; }
            double d = ll[i] - ll[best];
            /* tie: relative 1e-12 (degenerate pairs such as (1,2),(2,1) on a square) */
            double tol = 1e-12 * (ll[i] > ll[best] ? ll[i] : ll[best]);
            if (d < -tol) best = i;
            else if (fabs(d) <= tol) {
                if (mm[i] < mm[best] || (mm[i] == mm[best] && nn[i] < nn[best])) best = i;
            }
        }
        m_out[k] = mm[best]; n_out[k] = nn[best]; lambda_out[k] = ll[best];
        mm[best] = 0;
    }
    free(mm); free(nn); free(ll);
    return 0;
}

double orc_rect_mode(int m, int n, double Lx, double Ly, double x, double y)
{
    return 2.0 / sqrt(Lx * Ly) * sin(m * ORC_PI * x / Lx) * sin(n * ORC_PI * y / Ly);
}

/* ------------------------------------------------------------------------ */
/* 2. Modal oscillator coefficients (Eq. 13-14).           */
/*    omega^2 = (D lambda^2 + T0 lambda)/rho_m ; gamma = sigma0 + sigma1     */
/*    lambda with sigma0 = d1/(2 rho_m), sigma1 = d3/(2 rho_m) (reading R9:  */
/*    Eq. 14's sign).  rho_m = mass per unit length / area (reading R3).     */
/* ------------------------------------------------------------------------ */
void orc_omega_gamma(int N, const double *lambda, double D, double T0, double rho_m,
                     double sigma0, double sigma1, double *omega, double *gamma)
{
    for (int k = 0; k < N; ++k) {
        omega[k] = sqrt((D * lambda[k] * lambda[k] + T0 * lambda[k]) / rho_m);
        gamma[k] = sigma0 + sigma1 * lambda[k];
    }
}

/* tau (Eq. 4) */
double orc_tau_string(double E, double A, double L) { return E * A / (2.0 * L); }
double orc_tau_membrane(double E, double h, double Lx, double Ly, double nu)
{
    return E * h / (2.0 * Lx * Ly * (1.0 - nu * nu));
}

/* ------------------------------------------------------------------------ */
/* 3. von Karman operator and coupling coefficients                          */
/*    (Eq. 7; Eq. 10-11).                    */
/* ------------------------------------------------------------------------ */

/* L(f,g) = Lap f Lap g - Hess f : Hess g = f_xx g_yy + f_yy g_xx - 2 f_xy g_xy */
double orc_vk_operator(double fxx, double fyy, double fxy, double gxx, double gyy, double gxy)
{
    double lapf = fxx + fyy, lapg = gxx + gyy;
    double ddot = fxx * gxx + fyy * gyy + 2.0 * fxy * gxy; /* Hess f : Hess g */
    return lapf * lapg - ddot;
}

/* second derivatives of the unit-norm sine mode (m,n) at (x,y) */
static void rect_mode_hess(int m, int n, double Lx, double Ly, double x, double y,
                           double *fxx, double *fyy, double *fxy)
{
    double a = m * ORC_PI / Lx, b = n * ORC_PI / Ly, c = 2.0 / sqrt(Lx * Ly);
    *fxx = -a * a * c * sin(a * x) * sin(b * y);
    *fyy = -b * b * c * sin(a * x) * sin(b * y);
    *fxy = a * b * c * cos(a * x) * cos(b * y);
}

/* Brute-force Eq. 10: H^k_{ij} = int_S Psi_k L(Phi_i, Phi_j) dS by tensor-product
 * Gauss-Legendre quadrature of the 2-D integrand (nodes xg, weights wg on [-1,1],
 * ng points per axis, supplied by the caller).  Unit-norm modes: the
 * denominators of Eq. 10 are 1 (reading R6). */
double orc_H_quadrature(double Lx, double Ly, int mi, int ni, int mj, int nj, int mk, int nk,
                        int ng, const double *xg, const double *wg)
{
    double acc = 0.0;
    for (int a = 0; a < ng; ++a) {
        double x = 0.5 * Lx * (xg[a] + 1.0);
        for (int b = 0; b < ng; ++b) {
            double y = 0.5 * Ly * (xg[b] + 1.0);
            double ixx, iyy, ixy, jxx, jyy, jxy;
            rect_mode_hess(mi, ni, Lx, Ly, x, y, &ixx, &iyy, &ixy);
            rect_mode_hess(mj, nj, Lx, Ly, x, y, &jxx, &jyy, &jxy);
            double psi = orc_rect_mode(mk, nk, Lx, Ly, x, y);
            acc += wg[a] * wg[b] * psi * orc_vk_operator(ixx, iyy, ixy, jxx, jyy, jxy);
        }
    }
    return acc * 0.25 * Lx * Ly;
}

/* Brute-force Eq. 11: C^s_{ij} = int_S Phi_s L(Phi_i, Psi_j) dS, same quadrature.
 * Used only to check the identity H^k_{ij} = C^j_{ik}. */
double orc_C_quadrature(double Lx, double Ly, int ms, int ns, int mi, int ni, int mj, int nj,
                        int ng, const double *xg, const double *wg)
{
    /* same integrand shape: Phi_s * L(Phi_i, Psi_j) -- all three are sine modes */
    return orc_H_quadrature(Lx, Ly, mi, ni, mj, nj, ms, ns, ng, xg, wg);
}

/* Closed form of Eq. 10 for sine bases (derivation in DESIGN.md "H closed form").
 * J(k,c) = int_0^1 cos(k pi xi) sin(c pi xi) d xi = 2c / (pi (c^2 - k^2)) if k+c odd else 0. */
static double Jcs(int k, int c)
{
    if (k < 0) k = -k;
    if (((k + c) & 1) == 0) return 0.0;
    return 2.0 * c / (ORC_PI * ((double)c * c - (double)k * k));
}
static double sss(int a, int b, int c) { return 0.5 * (Jcs(a - b, c) - Jcs(a + b, c)); }
static double ccs(int a, int b, int c) { return 0.5 * (Jcs(a - b, c) + Jcs(a + b, c)); }

double orc_H_closed_entry(double Lx, double Ly, int mp, int np, int mq, int nq, int mn, int nn)
{
    double geom = 8.0 * pow(ORC_PI, 4) * pow(Lx * Ly, -2.5);
    double br = ((double)mp * mp * nq * nq + (double)np * np * mq * mq) * sss(mp, mq, mn) * sss(np, nq, nn)
              - 2.0 * (double)mp * np * mq * nq * ccs(mp, mq, mn) * ccs(np, nq, nn);
    return geom * br;
}

/* Full tensor H[n][p][q], row-major [Nphi][Nq][Nq]; transverse index set (mq,nq), in-plane
 * index set (mphi,nphi) (reading R5: Psi = sine products). */
void orc_H_closed(double Lx, double Ly, int Nq, const int *mq, const int *nq,
                  int Nphi, const int *mphi, const int *nphi, double *H)
{
    for (int n = 0; n < Nphi; ++n)
        for (int p = 0; p < Nq; ++p)
            for (int q = 0; q < Nq; ++q)
                H[((size_t)n * Nq + p) * Nq + q] =
                    orc_H_closed_entry(Lx, Ly, mq[p], nq[p], mq[q], nq[q], mphi[n], nphi[n]);
}

/* ------------------------------------------------------------------------ */
/* 4. Non-linear modal forces.                                               */
/* ------------------------------------------------------------------------ */

/* Eq. 8 under reading R2:
 *   S = sum_nu lambda_nu q_nu^2 ;  f_mu = c lambda_mu q_mu S,  c = tau / rho_m. */
void orc_tension_force(int N, const double *lambda, double c, const double *q, double *f)
{
    double S = 0.0;
    for (int nu = 0; nu < N; ++nu) S += lambda[nu] * q[nu] * q[nu];
    for (int mu = 0; mu < N; ++mu) f[mu] = c * lambda[mu] * q[mu] * S;
}

double orc_tension_S(int N, const double *lambda, const double *q)
{
    double S = 0.0;
    for (int nu = 0; nu < N; ++nu) S += lambda[nu] * q[nu] * q[nu];
    return S;
}

/* G_n(q) = sum_{p,q} H^n_{pq} q_p q_q  (first stage of Eq. 9) */
void orc_vk_G(int Nq, int Nphi, const double *H, const double *q, double *G)
{
    for (int n = 0; n < Nphi; ++n) {
        double acc = 0.0;
        for (int p = 0; p < Nq; ++p)
            for (int r = 0; r < Nq; ++r)
                acc += H[((size_t)n * Nq + p) * Nq + r] * q[p] * q[r];
        G[n] = acc;
    }
}

/* Eq. 9 in two stages, with C^s_{p,n} = H^n_{p,s}:
 *   eta_n = s_n G_n,   s_n = E / (2 rho zeta_n^4)
 *   f_s   = sum_n eta_n sum_p H^n_{p,s} q_p.
 * work: scratch of Nphi doubles. */
void orc_vk_force(int Nq, int Nphi, const double *H, const double *s, const double *q,
                  double *f, double *work)
{
    orc_vk_G(Nq, Nphi, H, q, work);
    for (int n = 0; n < Nphi; ++n) work[n] *= s[n];
    for (int k = 0; k < Nq; ++k) f[k] = 0.0;
    for (int n = 0; n < Nphi; ++n)
        for (int p = 0; p < Nq; ++p) {
            double e = work[n] * q[p];
            for (int k = 0; k < Nq; ++k)
                f[k] += H[((size_t)n * Nq + p) * Nq + k] * e;
        }
}

/* Eq. 9 as printed: one quintuple loop over (s; p,q,r,n) with separate tensors
 * Hq[n][q][r] and Cc[s][p][n]; scale[n] = E/(2 rho zeta_n^4). */
void orc_vk_force_naive(int Nq, int Nphi, const double *Hq, const double *Cc,
                        const double *scale, const double *q, double *f)
{
    for (int s = 0; s < Nq; ++s) {
        double acc = 0.0;
        for (int p = 0; p < Nq; ++p)
            for (int qq = 0; qq < Nq; ++qq)
                for (int r = 0; r < Nq; ++r)
                    for (int n = 0; n < Nphi; ++n)
                        acc += scale[n] * Hq[((size_t)n * Nq + qq) * Nq + r]
                             * Cc[((size_t)s * Nq + p) * Nphi + n] * q[p] * q[qq] * q[r];
        f[s] = acc;
    }
}

/* ------------------------------------------------------------------------ */
/* 5. Scheme coefficients.                                                   */
/* ------------------------------------------------------------------------ */

/* Stormer-Verlet, Eq. 21-23 as printed:
 *   r = 2T^2/(2+2 gamma T), g = r (2/T^2 - omega^2), p = r(-1/T^2 + 2 gamma/(2T)). */
void orc_sv_coeffs(int N, const double *omega, const double *gamma, double T,
                   double *g, double *p, double *r)
{
    for (int k = 0; k < N; ++k) {
        r[k] = 2.0 * T * T / (2.0 + 2.0 * gamma[k] * T);
        g[k] = r[k] * (2.0 / (T * T) - omega[k] * omega[k]);
        p[k] = r[k] * (-1.0 / (T * T) + 2.0 * gamma[k] / (2.0 * T));
    }
}

/* FTM / impulse invariance, Eq. 16-18, reading R7:
 *   a1 = -2 e^{-gamma T} cos(w~ T), a2 = e^{-2 gamma T},
 *   b1 = T e^{-gamma T} sin(w~ T)/w~   (per-unit-mass force, sampling period T),
 *   w~ = sqrt(omega^2 - gamma^2). */
void orc_ftm_coeffs(int N, const double *omega, const double *gamma, double T,
                    double *a1, double *a2, double *b1)
{
    for (int k = 0; k < N; ++k) {
        double wt = sqrt(omega[k] * omega[k] - gamma[k] * gamma[k]);
        a1[k] = -2.0 * exp(-gamma[k] * T) * cos(wt * T);
        a2[k] = exp(-2.0 * gamma[k] * T);
        b1[k] = T * exp(-gamma[k] * T) * sin(wt * T) / wt;
    }
}

/* ------------------------------------------------------------------------ */
/* 6. Time stepping (Eq. 19 / Eq. 20).                     */
/*    q^{n+1} = c1 q^n + c2 q^{n-1} + c3 (fext^n - fnl(q^n))                 */
/*    SV : (c1,c2,c3) = (g, p, r);  FTM : (-a1, -a2, b1) (reading R7).       */
/*    out[n] = sum_k w_k q_k^n for n = 0..n_steps-1 (reading R10).           */
/* ------------------------------------------------------------------------ */

enum { ORC_LINEAR = 0, ORC_TENSION = 1, ORC_VK = 2 };

typedef struct {
    int model;            /* ORC_LINEAR / ORC_TENSION / ORC_VK                       */
    int Nq, Nphi;         /* Nphi = 0 unless ORC_VK                                   */
    int batch, n_steps;
    int coeff_batch;      /* 1 = coefficient rows shared by all samples, else = batch */
    const double *c1, *c2, *c3;   /* [coeff_batch][Nq]                                */
    const double *w;              /* pickup weights [coeff_batch][Nq]                 */
    const double *lambda;         /* TENSION: [coeff_batch][Nq]                       */
    const double *nl_scale;       /* TENSION: tau/rho_m [coeff_batch]; VK: s_n [coeff_batch][Nphi] */
    const double *H;              /* VK: [Nphi][Nq][Nq], shared by the batch          */
    const double *q0, *qm1;       /* [batch][Nq] states at n = 0 and n = -1           */
    const double *fext;           /* optional [batch][n_steps] scalar signal, or NULL */
    const double *fext_gain;      /* optional [batch][Nq]                             */
    double *out;                  /* [batch][n_steps]                                 */
    int *first_bad;               /* [batch]: first n with a non-finite q^n, or -1    */
    double *traj;                 /* optional [batch][n_steps][Nq] full trajectory    */
    double *q_final;              /* optional [batch][2][Nq]: q^{n_steps-1} then q^{n_steps}          */
} orc_sim_args;

static void nl_force(const orc_sim_args *a, int cb, const double *q, double *f, double *work)
{
    int Nq = a->Nq;
    if (a->model == ORC_VK) {
        orc_vk_force(Nq, a->Nphi, a->H, a->nl_scale + (size_t)cb * a->Nphi, q, f, work);
    } else if (a->model == ORC_TENSION) {
        orc_tension_force(Nq, a->lambda + (size_t)cb * Nq, a->nl_scale[cb], q, f);
    } else {
        for (int k = 0; k < Nq; ++k) f[k] = 0.0;
    }
}

/* Simulate every sample.  q_final, if given, receives q^{n_steps-1} then q^{n_steps}
 * (the two states after the last recorded sample), so a run can be continued.
 * Returns the number of samples that went non-finite. */
int orc_simulate(const orc_sim_args *a)
{
    int Nq = a->Nq, nbad = 0;
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : nbad)
    for (int b = 0; b < a->batch; ++b) {
        int cb = a->coeff_batch == 1 ? 0 : b;
        const double *c1 = a->c1 + (size_t)cb * Nq, *c2 = a->c2 + (size_t)cb * Nq,
                     *c3 = a->c3 + (size_t)cb * Nq, *w = a->w + (size_t)cb * Nq;
        double *qn = (double *)malloc(sizeof(double) * Nq);
        double *qp = (double *)malloc(sizeof(double) * Nq);
        double *qx = (double *)malloc(sizeof(double) * Nq);
        double *f = (double *)malloc(sizeof(double) * Nq);
        double *work = (double *)malloc(sizeof(double) * (a->Nphi > 0 ? a->Nphi : 1));
        memcpy(qn, a->q0 + (size_t)b * Nq, sizeof(double) * Nq);
        memcpy(qp, a->qm1 + (size_t)b * Nq, sizeof(double) * Nq);
        int bad = -1;
        for (int n = 0; n < a->n_steps; ++n) {
            double o = 0.0;
            int finite = 1;
            for (int k = 0; k < Nq; ++k) {
                o += w[k] * qn[k];
                if (!isfinite(qn[k])) finite = 0;
            }
            a->out[(size_t)b * a->n_steps + n] = o;
            if (a->traj) memcpy(a->traj + ((size_t)b * a->n_steps + n) * Nq, qn, sizeof(double) * Nq);
            if (!finite && bad < 0) bad = n;
            nl_force(a, cb, qn, f, work);
            double fe = a->fext ? a->fext[(size_t)b * a->n_steps + n] : 0.0;
            for (int k = 0; k < Nq; ++k) {
                double fx = a->fext ? fe * a->fext_gain[(size_t)b * Nq + k] : 0.0;
                qx[k] = c1[k] * qn[k] + c2[k] * qp[k] + c3[k] * (fx - f[k]);
            }
            double *t = qp; qp = qn; qn = qx; qx = t;
        }
        if (a->q_final) {
            memcpy(a->q_final + ((size_t)b * 2 + 0) * Nq, qp, sizeof(double) * Nq);
            memcpy(a->q_final + ((size_t)b * 2 + 1) * Nq, qn, sizeof(double) * Nq);
        }
        if (a->first_bad) a->first_bad[b] = bad;
        if (bad >= 0) nbad += 1;
        free(qn); free(qp); free(qx); free(f); free(work);
    }
    return nbad;
}

/* ------------------------------------------------------------------------ */
/* 7. Discrete energy of the lossless SV scheme (reading R12):               */
/*   h^{n+1/2} = 1/2 sum ((q^{n+1}-q^n)/T)^2 + 1/2 sum omega^2 q^{n+1} q^n    */
/*             + V-product term:                                             */
/*       VK      : (E/(8 rho)) sum_n G_n(q^{n+1}) G_n(q^n) / zeta_n^4         */
/*                 = 1/4 sum_n s_n G_n(q^{n+1}) G_n(q^n)                      */
/*       TENSION : (tau/(4 rho_m)) S(q^{n+1}) S(q^n)                          */
/* traj: [n_steps][Nq] of ONE sample; energy: [n_steps-1].                    */
/* ------------------------------------------------------------------------ */
void orc_energy(int model, int Nq, int Nphi, int n_steps, double T, const double *omega,
                const double *lambda, const double *nl_scale, const double *H,
                const double *traj, double *energy)
{
    double *Ga = (double *)malloc(sizeof(double) * (Nphi > 0 ? Nphi : 1));
    double *Gb = (double *)malloc(sizeof(double) * (Nphi > 0 ? Nphi : 1));
    for (int n = 0; n + 1 < n_steps; ++n) {
        const double *qa = traj + (size_t)n * Nq, *qb = traj + (size_t)(n + 1) * Nq;
        double kin = 0.0, pot = 0.0, vnl = 0.0;
        for (int k = 0; k < Nq; ++k) {
            double v = (qb[k] - qa[k]) / T;
            kin += 0.5 * v * v;
            pot += 0.5 * omega[k] * omega[k] * qb[k] * qa[k];
        }
        if (model == ORC_VK) {
            orc_vk_G(Nq, Nphi, H, qa, Ga);
            orc_vk_G(Nq, Nphi, H, qb, Gb);
            for (int m = 0; m < Nphi; ++m) vnl += 0.25 * nl_scale[m] * Ga[m] * Gb[m];
        } else if (model == ORC_TENSION) {
            vnl = 0.25 * nl_scale[0] * orc_tension_S(Nq, lambda, qa) * orc_tension_S(Nq, lambda, qb);
        }
        energy[n] = kin + pot + vnl;
    }
    free(Ga); free(Gb);
}

/* Non-linear potential (reading R4): V = 1/4 sum_n s_n G_n^2 (VK), (c/4) S^2 (TENSION). */
double orc_potential_nl(int model, int Nq, int Nphi, const double *lambda, const double *nl_scale,
                        const double *H, const double *q)
{
    double v = 0.0;
    if (model == ORC_VK) {
        double *G = (double *)malloc(sizeof(double) * Nphi);
        orc_vk_G(Nq, Nphi, H, q, G);
        for (int n = 0; n < Nphi; ++n) v += 0.25 * nl_scale[n] * G[n] * G[n];
        free(G);
    } else if (model == ORC_TENSION) {
        double S = orc_tension_S(Nq, lambda, q);
        v = 0.25 * nl_scale[0] * S * S;
    }
    return v;
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
