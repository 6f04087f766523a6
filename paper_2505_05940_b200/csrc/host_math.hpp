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
