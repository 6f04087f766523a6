// host_math.hpp -- host-side (fp64) derivations of the product path: mode index sets,
// oscillator and scheme coefficients, the closed-form coupling tensor of the simply supported
// plate and the projection of the excitation bump (device layouts: flow_schedule.hpp, mma_schedule.hpp).  Independent of oracle/ (no shared code or tables).
#pragma once
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <string>
#include <vector>

namespace modal_host {

constexpr double PI = 3.141592653589793238462643383279502884;

struct ModeSet {
    std::vector<int> m, n;       // string: n[k] = 0
    std::vector<double> lambda;  // Laplacian eigenvalues (Eq. 2)
};

// Fixed string: Phi_m = sqrt(2/L) sin(m pi x/L), lambda_m = (m pi/L)^2.
inline ModeSet string_modes(double L, int N)
{
    ModeSet s;
    for (int m = 1; m <= N; ++m) {
        s.m.push_back(m); s.n.push_back(0);
        s.lambda.push_back((m * PI / L) * (m * PI / L));
    }
    return s;
}

inline double rect_lambda(int m, int n, double Lx, double Ly)
{
    const double a = m * PI / Lx, b = n * PI / Ly;
    return a * a + b * b;
}

// Simply supported rectangle: the N smallest lambda_{mn}, ascending, ties (relative 1e-12)
// ordered by (m, n).  Candidates: every (m,n) with lambda <= the N-th value of
// a bound that certainly holds N points; sorted, then near-equal runs re-ordered.
inline ModeSet rect_modes(double Lx, double Ly, int N)
{
    struct C { double l; int m, n; };
    // lambda(k,1), k = 1..N are N distinct points => the N-th smallest is <= lambda(N,1); same for (1,k)
    const double bound = std::min(rect_lambda(N, 1, Lx, Ly), rect_lambda(1, N, Lx, Ly)) * (1.0 + 1e-9);
    std::vector<C> c;
    for (int m = 1; rect_lambda(m, 1, Lx, Ly) <= bound; ++m)
        for (int n = 1; rect_lambda(m, n, Lx, Ly) <= bound; ++n) c.push_back({rect_lambda(m, n, Lx, Ly), m, n});
    std::sort(c.begin(), c.end(), [](const C &a, const C &b) {
        if (a.l != b.l) return a.l < b.l;
        return a.m != b.m ? a.m < b.m : a.n < b.n;
    });
    for (size_t i = 0; i < c.size();) {       // runs of numerically equal lambda
        size_t j = i + 1;
        while (j < c.size() && c[j].l - c[i].l <= 1e-12 * c[j].l) ++j;
        std::sort(c.begin() + i, c.begin() + j,
                  [](const C &a, const C &b) { return a.m != b.m ? a.m < b.m : a.n < b.n; });
        i = j;
    }
    ModeSet s;
    for (int k = 0; k < N && k < (int)c.size(); ++k) {
        s.m.push_back(c[k].m); s.n.push_back(c[k].n); s.lambda.push_back(c[k].l);
    }
    return s;
}

inline double plate_D(double E, double h, double nu) { return E * h * h * h / (12.0 * (1.0 - nu * nu)); }

// PAPER.md:133-136, Eq. 13-14
inline void omega_sigma(const std::vector<double> &lambda, double D, double T0, double rho_m,
                        double sigma0, double sigma1, double *omega, double *sigma)
{
    for (size_t k = 0; k < lambda.size(); ++k) {
        omega[k] = std::sqrt((D * lambda[k] * lambda[k] + T0 * lambda[k]) / rho_m);
        sigma[k] = sigma0 + sigma1 * lambda[k];
    }
}

// Reading R11: modes the explicit scheme cannot carry are masked.
inline bool mode_active(int scheme, double omega, double sigma, double T)
{
    if (scheme == 0) return omega * T < 1.9;
    const double w2 = omega * omega - sigma * sigma;
    return std::sqrt(w2 > 0 ? w2 : 0.0) < 0.95 * PI / T;
}

struct StepCoeffs { double kv, kq, r, astart; };
// Delta-form coefficients of the two schemes (kernels.cuh header comment).
inline StepCoeffs step_coeffs(int scheme, double omega, double sigma, double T)
{
    StepCoeffs c;
    if (scheme == 0) {  // Stormer-Verlet, Eq. 21-23
        c.r = T * T / (1.0 + sigma * T);
        c.kv = (1.0 - sigma * T) / (1.0 + sigma * T);
        c.kq = c.r * omega * omega;
    } else {            // FTM / impulse invariance, Eq. 16-18 (reading R7)
        const double wt = std::sqrt(omega * omega - sigma * sigma);
        const double e = std::exp(-sigma * T);
        c.kv = e * e;
        // 1 + a1 + a2 = (1 - e)^2 + 2 e (1 - cos) = (1-e)^2 + 4 e sin^2(wt T / 2): no cancellation
        const double sh = std::sin(0.5 * wt * T);
        c.kq = (1.0 - e) * (1.0 - e) + 4.0 * e * sh * sh;
        c.r = T * e * std::sin(wt * T) / wt;
    }
    c.astart = 0.5 * T * T * omega * omega;   // reading R8: v^0 = (T^2/2)(omega^2 q^0 + fnl(q^0))
    return c;
}

// ---- coupling coefficients of the simply supported plate (Eq. 10) -------
// F(j) = int_0^1 sin(j pi x) dx
inline double Fint(int j) { return (j & 1) ? 2.0 / (j * PI) : 0.0; }
// int_0^1 sin(a pi x) sin(b pi x) sin(c pi x) dx   (product-to-sum, 4 terms)
inline double S3(int a, int b, int c)
{
    return 0.25 * (Fint(a + b - c) + Fint(a - b + c) + Fint(-a + b + c) - Fint(a + b + c));
}
// int_0^1 cos(a pi x) cos(b pi x) sin(c pi x) dx
inline double C3(int a, int b, int c)
{
    return 0.25 * (Fint(c + a + b) + Fint(c - a - b) + Fint(c + a - b) + Fint(c - a + b));
}
// Integer bracket: H^n_pq = 8 pi^4 (Lx Ly)^(-5/2) * bracket
inline double H_bracket(int mp, int np, int mq, int nq, int mn, int nn)
{
    const double A = (double)mp * mp * nq * nq + (double)np * np * mq * mq;
    const double B = 2.0 * mp * np * (double)mq * nq;
    return A * S3(mp, mq, mn) * S3(np, nq, nn) - B * C3(mp, mq, mn) * C3(np, nq, nn);
}
inline double H_geom(double Lx, double Ly) { return 8.0 * std::pow(PI, 4) * std::pow(Lx * Ly, -2.5); }

// ---- in-plane basis, reading R16: clamped-plate Airy modes by Rayleigh-Ritz ---------
// Lap Lap Psi = zeta^4 Psi with Psi = dPsi/dn = 0 on the edges ("a Galerkin type approach").  Trial space
// T_i(x/Lx) T_j(y/Ly), T_i(s) = sin(pi s) sin(i pi s) = (cos((i-1) pi s) - cos((i+1) pi s)) / 2: every integral is a finite sum of
//     I(u, v) = int_0^1 cos(u pi s) cos(v pi s) ds = 1 (u = v = 0), 1/2 (u = v > 0), 0 otherwise,
// so the matrices are exact; the generalised eigenproblem is solved per symmetry class (T_i is even about s = 1/2 for odd i, odd for
// even i; the four (x, y) classes do not couple) by Cholesky reduction + cyclic Jacobi.  The oracle does the same problem with
// Gauss-Legendre quadrature and LAPACK (oracle/oracle.py airy_ritz_basis), sharing no code.
inline double cosI(int u, int v) { u = u < 0 ? -u : u; v = v < 0 ? -v : v; return u != v ? 0.0 : (u == 0 ? 1.0 : 0.5); }
// T_i = sum_u tau(i,u) cos(u pi s): tau(i, i-1) = 1/2, tau(i, i+1) = -1/2
struct RitzTrial {
    int nt;
    explicit RitzTrial(int n) : nt(n) {}
    template <class F> void terms(int i, F f) const { f(i - 1, 0.5); f(i + 1, -0.5); }       // (u, tau)
    double A(int i, int j, int order) const {       // order 0: int T_i T_j; 1: int T_i' T_j'; 2: int T_i'' T_j''
        double acc = 0;
        terms(i, [&](int u, double a) { terms(j, [&](int v, double b) {
            if (order == 0) acc += a * b * cosI(u, v);
            else if (order == 1) acc += a * b * (u * PI) * (v * PI) * (u == v && u > 0 ? 0.5 : 0.0);     // int sin sin
            else acc += a * b * std::pow(u * PI, 2) * std::pow(v * PI, 2) * cosI(u, v);
        }); });
        return acc;
    }
    double SS(int i, int a, int b) const {          // int T_i sin(a pi s) sin(b pi s)
        double acc = 0;
        terms(i, [&](int u, double t) { acc += 0.5 * t * (cosI(u, a - b) - cosI(u, a + b)); });
        return acc;
    }
    double CC(int i, int a, int b) const {          // int T_i cos(a pi s) cos(b pi s)
        double acc = 0;
        terms(i, [&](int u, double t) { acc += 0.5 * t * (cosI(u, a - b) + cosI(u, a + b)); });
        return acc;
    }
};

// Symmetric generalised eigenproblem K c = lam M c (M positive definite), n x n row-major: eigenvalues ascending in lam,
// M-orthonormal eigenvectors in the columns of V.  Cholesky M = L L^T, C = L^-1 K L^-T, cyclic Jacobi on C.
inline bool sym_gen_eig(int n, std::vector<double> K, std::vector<double> M, std::vector<double> &lam, std::vector<double> &V)
{
    std::vector<double> L((size_t)n * n, 0.0);
    for (int i = 0; i < n; ++i)
        for (int j = 0; j <= i; ++j) {
            double s = M[(size_t)i * n + j];
            for (int k = 0; k < j; ++k) s -= L[(size_t)i * n + k] * L[(size_t)j * n + k];
            if (i == j) { if (!(s > 0)) return false; L[(size_t)i * n + i] = std::sqrt(s); }
            else L[(size_t)i * n + j] = s / L[(size_t)j * n + j];
        }
    // C = L^-1 K L^-T : solve L X = K (columns), then L Y^T = X^T
    std::vector<double> X((size_t)n * n), C((size_t)n * n);
    for (int c = 0; c < n; ++c)
        for (int i = 0; i < n; ++i) {
            double s = K[(size_t)i * n + c];
            for (int k = 0; k < i; ++k) s -= L[(size_t)i * n + k] * X[(size_t)k * n + c];
            X[(size_t)i * n + c] = s / L[(size_t)i * n + i];
        }
    for (int r = 0; r < n; ++r)
        for (int i = 0; i < n; ++i) {
            double s = X[(size_t)r * n + i];
            for (int k = 0; k < i; ++k) s -= L[(size_t)i * n + k] * C[(size_t)r * n + k];
            C[(size_t)r * n + i] = s / L[(size_t)i * n + i];
        }
    std::vector<double> Q((size_t)n * n, 0.0);
    for (int i = 0; i < n; ++i) Q[(size_t)i * n + i] = 1.0;
    for (int sweep = 0; sweep < 60; ++sweep) {
        double off = 0, diag = 0;
        for (int i = 0; i < n; ++i) { diag += C[(size_t)i * n + i] * C[(size_t)i * n + i]; for (int j = 0; j < i; ++j) off += C[(size_t)i * n + j] * C[(size_t)i * n + j]; }
        if (off <= 1e-30 * diag) break;
        for (int p = 0; p < n - 1; ++p)
            for (int q = p + 1; q < n; ++q) {
                const double apq = C[(size_t)p * n + q];
                if (std::fabs(apq) < 1e-300) continue;
                const double theta = (C[(size_t)q * n + q] - C[(size_t)p * n + p]) / (2.0 * apq);
                const double t = (theta >= 0 ? 1.0 : -1.0) / (std::fabs(theta) + std::sqrt(theta * theta + 1.0));
                const double cs = 1.0 / std::sqrt(t * t + 1.0), sn = t * cs;
                for (int k = 0; k < n; ++k) {
                    const double ckp = C[(size_t)k * n + p], ckq = C[(size_t)k * n + q];
                    C[(size_t)k * n + p] = cs * ckp - sn * ckq; C[(size_t)k * n + q] = sn * ckp + cs * ckq;
                }
                for (int k = 0; k < n; ++k) {
                    const double cpk = C[(size_t)p * n + k], cqk = C[(size_t)q * n + k];
                    C[(size_t)p * n + k] = cs * cpk - sn * cqk; C[(size_t)q * n + k] = sn * cpk + cs * cqk;
                }
                for (int k = 0; k < n; ++k) {
                    const double qkp = Q[(size_t)k * n + p], qkq = Q[(size_t)k * n + q];
                    Q[(size_t)k * n + p] = cs * qkp - sn * qkq; Q[(size_t)k * n + q] = sn * qkp + cs * qkq;
                }
            }
    }
    std::vector<int> order(n);
    for (int i = 0; i < n; ++i) order[i] = i;
    std::sort(order.begin(), order.end(), [&](int a, int b) { return C[(size_t)a * n + a] < C[(size_t)b * n + b]; });
    lam.resize(n); V.assign((size_t)n * n, 0.0);
    for (int e = 0; e < n; ++e) {
        const int src = order[e];
        lam[e] = C[(size_t)src * n + src];
        // v = L^-T q
        for (int i = n - 1; i >= 0; --i) {
            double s = Q[(size_t)i * n + src];
            for (int k = i + 1; k < n; ++k) s -= L[(size_t)k * n + i] * V[(size_t)k * n + e];
            V[(size_t)i * n + e] = s / L[(size_t)i * n + i];
        }
    }
    return true;
}

struct AiryRitz {
    int nt = 0;
    std::vector<double> zeta4;             // [n_phi] ascending
    std::vector<double> c;                 // [n_phi][nt][nt], Psi_n = sum c[n][i-1][j-1] T_i(x/Lx) T_j(y/Ly), unit L2 norm, largest coefficient positive
};

inline bool airy_ritz_basis(double Lx, double Ly, int n_phi, int nt, AiryRitz &out)
{
    const RitzTrial T(nt);
    struct Mode { double z4; std::vector<double> c; };
    std::vector<Mode> all;
    for (int px = 0; px < 2; ++px)
        for (int py = 0; py < 2; ++py) {
            std::vector<int> ix, iy;                         // i odd (px = 0: even about the middle) or even
            for (int i = 1; i <= nt; ++i) { if ((i & 1) == (px ? 0 : 1)) ix.push_back(i); if ((i & 1) == (py ? 0 : 1)) iy.push_back(i); }
            const int nx = (int)ix.size(), ny = (int)iy.size(), n = nx * ny;
            if (n == 0) continue;
            std::vector<double> K((size_t)n * n), M((size_t)n * n);
            for (int a = 0; a < nx; ++a) for (int b = 0; b < ny; ++b)
                for (int a2 = 0; a2 < nx; ++a2) for (int b2 = 0; b2 < ny; ++b2) {
                    const double x0 = T.A(ix[a], ix[a2], 0), x1 = T.A(ix[a], ix[a2], 1), x2 = T.A(ix[a], ix[a2], 2);
                    const double y0 = T.A(iy[b], iy[b2], 0), y1 = T.A(iy[b], iy[b2], 1), y2 = T.A(iy[b], iy[b2], 2);
                    const size_t o = (size_t)(a * ny + b) * n + (a2 * ny + b2);
                    M[o] = Lx * Ly * x0 * y0;
                    K[o] = Lx * Ly * (x2 * y0 / std::pow(Lx, 4) + 2.0 * x1 * y1 / (Lx * Lx * Ly * Ly) + x0 * y2 / std::pow(Ly, 4));
                }
            std::vector<double> lam, V;
            if (!sym_gen_eig(n, K, M, lam, V)) return false;
            const int keep = std::min(n, n_phi);
            for (int e = 0; e < keep; ++e) {
                Mode m; m.z4 = lam[e]; m.c.assign((size_t)nt * nt, 0.0);
                for (int a = 0; a < nx; ++a) for (int b = 0; b < ny; ++b) m.c[(size_t)(ix[a] - 1) * nt + (iy[b] - 1)] = V[(size_t)(a * ny + b) * n + e];
                all.push_back(std::move(m));
            }
        }
    if ((int)all.size() < n_phi) return false;
    std::stable_sort(all.begin(), all.end(), [](const Mode &a, const Mode &b) { return a.z4 < b.z4; });
    out.nt = nt; out.zeta4.resize(n_phi); out.c.assign((size_t)n_phi * nt * nt, 0.0);
    for (int n = 0; n < n_phi; ++n) {
        out.zeta4[n] = all[n].z4;
        size_t k = 0;
        for (size_t x = 1; x < all[n].c.size(); ++x) if (std::fabs(all[n].c[x]) > std::fabs(all[n].c[k])) k = x;
        const double sg = all[n].c[k] < 0 ? -1.0 : 1.0;
        for (size_t x = 0; x < all[n].c.size(); ++x) out.c[(size_t)n * nt * nt + x] = sg * all[n].c[x];
    }
    return true;
}

// H^n_pq = int Psi_n L(Phi_p, Phi_q) dS for sine transverse modes p = (mp, np), q = (mq, nq) (Eq. 10, Eq. 7), closed form:
//   H = 4 [ (a_xp^2 a_yq^2 + a_yp^2 a_xq^2) sum_ij c_ij SS_i(mp, mq) SS_j(np, nq) - 2 a_xp a_yp a_xq a_yq sum_ij c_ij CC_i(mp, mq) CC_j(np, nq) ]
// with a_x = m pi / Lx, a_y = n pi / Ly.  SS_i(a, b) and CC_i(a, b) vanish unless i +- 1 is |a - b| or a + b: at most four i (and j) per entry.
inline double airy_ritz_H_entry(int nt, const double *c /*[nt][nt]*/, double Lx, double Ly, int mp, int np, int mq, int nq)
{
    const RitzTrial T(nt);
    auto cand = [&](int a, int b, int (&out)[4]) {
        const int u[2] = {a > b ? a - b : b - a, a + b};
        int cnt = 0;
        for (int x = 0; x < 2; ++x)
            for (int d = -1; d <= 1; d += 2) {
                const int i = u[x] + d;
                bool dup = false;
                for (int y = 0; y < cnt; ++y) dup |= out[y] == i;
                if (i >= 1 && i <= nt && !dup) out[cnt++] = i;
            }
        return cnt;
    };
    int ii[4], jj[4];
    const int ni = cand(mp, mq, ii), nj = cand(np, nq, jj);
    double t1 = 0, t2 = 0;
    for (int x = 0; x < ni; ++x) {
        const double sx = T.SS(ii[x], mp, mq), cx = T.CC(ii[x], mp, mq);
        for (int y = 0; y < nj; ++y) {
            const double cij = c[(size_t)(ii[x] - 1) * nt + (jj[y] - 1)];
            t1 += cij * sx * T.SS(jj[y], np, nq);
            t2 += cij * cx * T.CC(jj[y], np, nq);
        }
    }
    const double axp = mp * PI / Lx, ayp = np * PI / Ly, axq = mq * PI / Lx, ayq = nq * PI / Ly;
    return 4.0 * ((axp * axp * ayq * ayq + ayp * ayp * axq * axq) * t1 - 2.0 * axp * ayp * axq * ayq * t2);
}

// ---- excitation projection (reading R13) -------------------------------------------------
// Gauss-Legendre nodes on [-1,1] by Newton iteration on P_n.
inline void gauss_legendre(int n, std::vector<double> &x, std::vector<double> &w)
{
    x.resize(n); w.resize(n);
    for (int i = 0; i < (n + 1) / 2; ++i) {
        double z = std::cos(PI * (i + 0.75) / (n + 0.5)), pp = 0;
        for (int it = 0; it < 100; ++it) {
            double p1 = 1.0, p2 = 0.0;
            for (int j = 1; j <= n; ++j) { const double p3 = p2; p2 = p1; p1 = ((2.0 * j - 1.0) * z * p2 - (j - 1.0) * p3) / j; }
            pp = n * (z * p1 - p2) / (z * z - 1.0);
            const double dz = p1 / pp;
            z -= dz;
            if (std::fabs(dz) < 1e-15) break;
        }
        x[i] = -z; x[n - 1 - i] = z;
        w[i] = w[n - 1 - i] = 2.0 / ((1.0 - z * z) * pp * pp);
    }
}

// q0_k = int_disc (A/2)(1 + cos(2 pi r/W)) Phi_k dS ; polar rule: Gauss-Legendre in r, trapezoid in theta
inline void project_bump_rect(const ModeSet &ms, double Lx, double Ly, double x0, double y0,
                              double W, double A, double *q0)
{
    const int nr = 80, nth = 192;
    std::vector<double> xr, wr;
    gauss_legendre(nr, xr, wr);
    const double c = 2.0 / std::sqrt(Lx * Ly);
    const size_t N = ms.m.size();
    int Mx = 1, My = 1;
    for (size_t k = 0; k < N; ++k) { Mx = std::max(Mx, ms.m[k]); My = std::max(My, ms.n[k]); }
    std::vector<double> acc(N, 0.0), sx(Mx + 1), sy(My + 1);
    for (int i = 0; i < nr; ++i) {
        const double r = 0.25 * W * (xr[i] + 1.0);
        const double wt = 0.25 * W * wr[i] * r * 0.5 * A * (1.0 + std::cos(2.0 * PI * r / W)) * (2.0 * PI / nth);
        for (int j = 0; j < nth; ++j) {
            const double th = 2.0 * PI * j / nth;
            const double x = x0 + r * std::cos(th), y = y0 + r * std::sin(th);
            // sin(m a) for m = 0..M by the three-term recurrence s_{m+1} = 2 cos(a) s_m - s_{m-1}
            const double ax = PI * x / Lx, ay = PI * y / Ly, cx2 = 2.0 * std::cos(ax), cy2 = 2.0 * std::cos(ay);
            sx[0] = 0.0; sx[1] = std::sin(ax);
            for (int m = 1; m < Mx; ++m) sx[m + 1] = cx2 * sx[m] - sx[m - 1];
            sy[0] = 0.0; sy[1] = std::sin(ay);
            for (int m = 1; m < My; ++m) sy[m + 1] = cy2 * sy[m] - sy[m - 1];
            for (size_t k = 0; k < N; ++k) acc[k] += wt * sx[ms.m[k]] * sy[ms.n[k]];
        }
    }
    for (size_t k = 0; k < N; ++k) q0[k] = c * acc[k];
}

inline void project_bump_string(int N, double L, double x0, double W, double A, double *q0)
{
    const int ng = 200;
    std::vector<double> xg, wg;
    gauss_legendre(ng, xg, wg);
    for (int m = 1; m <= N; ++m) {
        double acc = 0.0;
        for (int i = 0; i < ng; ++i) {
            const double x = x0 + 0.5 * W * xg[i];
            acc += 0.5 * W * wg[i] * 0.5 * A * (1.0 + std::cos(2.0 * PI * (x - x0) / W)) * std::sin(m * PI * x / L);
        }
        q0[m - 1] = std::sqrt(2.0 / L) * acc;
    }
}

}  // namespace modal_host
