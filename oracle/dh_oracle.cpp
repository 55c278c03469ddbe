// =====================================================================================
// dh_oracle.cpp -- CPU ORACLE for the diffHydro coupled step and its adjoint.
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It
// shares no code, header, table or helper with the CUDA path (paper_2502_02294_b200/).
//
// What it is: the scheme of Horowitz & Lukic (arXiv 2502.02294), written out step by
// step in fp64 with plain loops, in the paper's order and notation, with the readings
// R1..R27 of SURVEY.md section 8(c) / DESIGN.md where the paper is silent or garbled.
// Every function cites the PAPER.md passage it follows.  OpenMP pragmas only spread
// independent pencils / particles / FFT lines over cores; they change no arithmetic.
//
// Contents
//   * forward:  sweep (relaxing TVD, Eq. 9-18), CIC deposit / gather
//               (PAPER.md:71, :244), FFT Poisson solve with spectral gradient (PAPER.md:71,
//               :83), kick-drift (Eq. 2-3), Strang ordering,
//               CFL maximum (Eq. 19-20).
//   * JVP:      the SAME templated forward code instantiated with a dual number
//               (value, derivative) scalar -- exact to round-off, no derivation.
//   * VJP:      hand-written reverse pass, statement by statement the transpose of the
//               forward (PAPER.md:198-206 describes reverse-mode replay of the primitives).
//
// Pins (tests/, -m "not gpu"): exact Riemann solution of the 1-D Sod tube, uniform-state
// preservation, conservation to round-off, axis symmetry, second-order convergence of a
// sound wave, limiter identities, single-mode Poisson vs its analytic force, own FFT vs
// numpy.fft, CIC mass/affine/adjoint-pair/no-self-force identities, EdS step factors,
// Zel'dovich pancake, Hubble-drag/adiabatic factors, cold-gas tracking of DM, JVP vs
// central finite differences, <Jv,w> = <v,J^T w>.
// "parity unpinned": the whole nonlinear coupled multi-step run has no printed values in
// the paper; it is trusted on the strength of the component pins above.
// =====================================================================================
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>
#include <algorithm>

#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ------------------------------------------------------------------ dual numbers ----
// value + one directional derivative; used to obtain J*v from the forward code itself.
struct Dual {
    double v, d;
    Dual() : v(0), d(0) {}
    Dual(double v_) : v(v_), d(0) {}
    Dual(double v_, double d_) : v(v_), d(d_) {}
};
inline Dual operator+(Dual a, Dual b) { return Dual(a.v + b.v, a.d + b.d); }
inline Dual operator-(Dual a, Dual b) { return Dual(a.v - b.v, a.d - b.d); }
inline Dual operator-(Dual a) { return Dual(-a.v, -a.d); }
inline Dual operator*(Dual a, Dual b) { return Dual(a.v * b.v, a.d * b.v + a.v * b.d); }
inline Dual operator/(Dual a, Dual b) {
    double q = a.v / b.v;
    return Dual(q, (a.d - q * b.d) / b.v);
}
inline Dual& operator+=(Dual& a, Dual b) { a = a + b; return a; }
inline Dual& operator-=(Dual& a, Dual b) { a = a - b; return a; }

inline double val(double x) { return x; }
inline double val(Dual x) { return x.v; }
inline double sqrt_(double x) { return std::sqrt(x); }
inline Dual sqrt_(Dual x) { double s = std::sqrt(x.v); return Dual(s, x.d / (2.0 * s)); }
// d|v|/dv = sign(v), sign(0) = 0  (R26)
inline double abs_(double x) { return std::fabs(x); }
inline Dual abs_(Dual x) {
    double s = (x.v > 0.0) - (x.v < 0.0);
    return Dual(std::fabs(x.v), s * x.d);
}
// e+ = max(e, floor); derivative 0 on the floored branch and at the switching point (R17, R26)
inline double floor_at(double e, double fl) { return e > fl ? e : fl; }
inline Dual floor_at(Dual e, double fl) { return e.v > fl ? e : Dual(fl, 0.0); }

// ---------------------------------------------------------------------- limiter -----
// PAPER.md:144-150, Eq. 18: "altered Van Leer" = harmonic mean 2ab/(a+b+eps).
// Reading R8: gated to ab > 0 (else 0), eps enters as sign(a)*eps so phi(-a,-b) = -phi(a,b).
template <class T>
inline T limiter(T a, T b, double eps) {
    if (val(a) * val(b) > 0.0) {
        double s = val(a) > 0.0 ? eps : -eps;
        return T(2.0) * a * b / (a + b + T(s));
    }
    return T(0.0);
}
// partial derivatives of the limiter (both 0 when ab <= 0)
inline void limiter_grad(double a, double b, double eps, double& da, double& db) {
    if (a * b > 0.0) {
        double s = a > 0.0 ? eps : -eps;
        double den = a + b + s;
        da = 2.0 * b * (b + s) / (den * den);
        db = 2.0 * a * (a + s) / (den * den);
    } else {
        da = 0.0; db = 0.0;
    }
}

// ------------------------------------------------------------- cell primitives ------
// One cell of one pencil: conserved u = (rho, m_n, m_t1, m_t2, eps) with m_n the momentum
// component along the sweep direction.  PAPER.md:95-101 (Eq. 8 state and flux vector, with
// R3: pressure in the normal momentum flux), PAPER.md:89 (EOS p=(gamma-1) rho e),
// PAPER.md:117 (freezing speed c = |v| + c_s, per cell: R11), R4 (F^R=(cU+F)/2, F^L=(cU-F)/2).
template <class T>
struct Prim {
    T c;          // freezing speed
    T FR[5];      // right-moving flux
    T FL[5];      // left-moving flux
};

template <class T>
inline Prim<T> prim(const T u[5], T gamma, double e_floor) {
    Prim<T> P;
    T rho = u[0], mn = u[1], mt1 = u[2], mt2 = u[3], eps = u[4];
    T v = mn / rho;                                                  // v~ = m_d / rho
    T e = eps / rho - (mn * mn + mt1 * mt1 + mt2 * mt2) / (T(2.0) * rho * rho);
    T ep = floor_at(e, e_floor);                                     // R17
    T p = (gamma - T(1.0)) * rho * ep;
    T cs = sqrt_(gamma * (gamma - T(1.0)) * ep);                     // c~_s = sqrt(gamma p/rho)
    P.c = abs_(v) + cs;
    T F[5];
    F[0] = mn;
    F[1] = mn * v + p;
    F[2] = mt1 * v;
    F[3] = mt2 * v;
    F[4] = (eps + p) * v;
    for (int k = 0; k < 5; ++k) {
        P.FR[k] = (P.c * u[k] + F[k]) / T(2.0);
        P.FL[k] = (P.c * u[k] - F[k]) / T(2.0);
    }
    return P;
}

// transpose of prim(): given cotangents of FR, FL add the cotangent of u and of gamma.
inline void prim_vjp(const double u[5], double gamma, double e_floor,
                     const double FRb[5], const double FLb[5],
                     double ub[5], double& gamma_b) {
    double rho = u[0], mn = u[1], mt1 = u[2], mt2 = u[3], eps = u[4];
    double v = mn / rho;
    double m2 = mn * mn + mt1 * mt1 + mt2 * mt2;
    double e = eps / rho - m2 / (2.0 * rho * rho);
    double ep = e > e_floor ? e : e_floor;
    double p = (gamma - 1.0) * rho * ep;
    double cs = std::sqrt(gamma * (gamma - 1.0) * ep);
    double c = std::fabs(v) + cs;

    // FR = (c u + F)/2, FL = (c u - F)/2
    double cub[5], Fb[5];
    for (int k = 0; k < 5; ++k) {
        cub[k] = 0.5 * (FRb[k] + FLb[k]);
        Fb[k] = 0.5 * (FRb[k] - FLb[k]);
    }
    double cb = 0.0;
    for (int k = 0; k < 5; ++k) { cb += cub[k] * u[k]; ub[k] += c * cub[k]; }
    // F = (mn, mn v + p, mt1 v, mt2 v, (eps+p) v)
    double mnb = Fb[0] + Fb[1] * v;
    double vb = Fb[1] * mn + Fb[2] * mt1 + Fb[3] * mt2 + Fb[4] * (eps + p);
    double pb = Fb[1] + Fb[4] * v;
    double mt1b = Fb[2] * v;
    double mt2b = Fb[3] * v;
    double epsb = Fb[4] * v;
    // c = |v| + cs
    double sgn = (v > 0.0) - (v < 0.0);
    vb += sgn * cb;
    double csb = cb;
    // cs = sqrt(gamma (gamma-1) ep)
    double epb = csb * gamma * (gamma - 1.0) / (2.0 * cs);
    gamma_b += csb * (2.0 * gamma - 1.0) * ep / (2.0 * cs);
    // p = (gamma-1) rho ep
    gamma_b += pb * rho * ep;
    double rhob = pb * (gamma - 1.0) * ep;
    epb += pb * (gamma - 1.0) * rho;
    // ep = max(e, floor)
    double eb = e > e_floor ? epb : 0.0;
    // e = eps/rho - m2/(2 rho^2)
    epsb += eb / rho;
    rhob += eb * (-eps / (rho * rho) + m2 / (rho * rho * rho));
    mnb += -eb * mn / (rho * rho);
    mt1b += -eb * mt1 / (rho * rho);
    mt2b += -eb * mt2 / (rho * rho);
    // v = mn / rho
    mnb += vb / rho;
    rhob += -vb * mn / (rho * rho);

    ub[0] += rhob; ub[1] += mnb; ub[2] += mt1b; ub[3] += mt2b; ub[4] += epsb;
}

inline int wrapi(int i, int n) { i %= n; return i < 0 ? i + n : i; }

// ------------------------------------------------------------------ 1-D sweep -------
// SWEEP_d on one periodic pencil of n cells.  u[k][i], k = (rho, m_n, m_t1, m_t2, eps).
//   Stage A (Eq. 12; first-order upwind Eq. 14 per wave family, R6/R7):
//       Phi_{i+1/2} = FR_i - FL_{i+1};  u*_i = u_i - (lam/2)(Phi_{i+1/2}-Phi_{i-1/2}) + (kap/2) S(u_i,g_i)
//   Stage B (Eq. 13 with second-order TVD fluxes Eq. 15-18):
//       PhiR_{i+1/2} = FR*_i     + phi((FR*_i - FR*_{i-1})/2, (FR*_{i+1} - FR*_i)/2)
//       PhiL_{i+1/2} = FL*_{i+1} - phi((FL*_{i+1} - FL*_i)/2, (FL*_{i+2} - FL*_{i+1})/2)
//       u'_i = u_i - lam (Phi*_{i+1/2} - Phi*_{i-1/2}) + kap S(u*_i, g_i)
//   Gravity source S(u,g) = (0, rho g, 0, 0, m_n g)   (S_g of Eq. 8; R2: S_e = 0)
//   lam = dtau/dx, kap = int dt/a (key identity of SURVEY.md 8; R15).
//   cmax = max_i c_i of the INPUT state (Eq. 19-20; R10).
template <class T>
void sweep_pencil(int n, const std::vector<T>* u, const T* g, T lam, T kap, T gamma,
                  double e_floor, double lim_eps, std::vector<T>* out, double* cmax) {
    std::vector<Prim<T>> P(n), Ps(n);
    std::vector<T> us[5];
    std::vector<T> Phi[5], Phis[5];
    for (int k = 0; k < 5; ++k) { us[k].resize(n); Phi[k].resize(n); Phis[k].resize(n); }
    double cm = 0.0;
    for (int i = 0; i < n; ++i) {
        T ui[5] = {u[0][i], u[1][i], u[2][i], u[3][i], u[4][i]};
        P[i] = prim(ui, gamma, e_floor);
        cm = std::max(cm, val(P[i].c));
    }
    if (cmax) *cmax = cm;
    // Stage A
    for (int i = 0; i < n; ++i) {
        int ip = wrapi(i + 1, n);
        for (int k = 0; k < 5; ++k) Phi[k][i] = P[i].FR[k] - P[ip].FL[k];       // Phi_{i+1/2}
    }
    for (int i = 0; i < n; ++i) {
        int im = wrapi(i - 1, n);
        T gi = g ? g[i] : T(0.0);
        T S[5] = {T(0.0), u[0][i] * gi, T(0.0), T(0.0), u[1][i] * gi};
        for (int k = 0; k < 5; ++k)
            us[k][i] = u[k][i] - (lam / T(2.0)) * (Phi[k][i] - Phi[k][im]) + (kap / T(2.0)) * S[k];
    }
    // Stage B
    for (int i = 0; i < n; ++i) {
        T ui[5] = {us[0][i], us[1][i], us[2][i], us[3][i], us[4][i]};
        Ps[i] = prim(ui, gamma, e_floor);
    }
    for (int i = 0; i < n; ++i) {
        int im = wrapi(i - 1, n), ip = wrapi(i + 1, n), ipp = wrapi(i + 2, n);
        for (int k = 0; k < 5; ++k) {
            T PhiR = Ps[i].FR[k] + limiter((Ps[i].FR[k] - Ps[im].FR[k]) / T(2.0),
                                           (Ps[ip].FR[k] - Ps[i].FR[k]) / T(2.0), lim_eps);
            T PhiL = Ps[ip].FL[k] - limiter((Ps[ip].FL[k] - Ps[i].FL[k]) / T(2.0),
                                            (Ps[ipp].FL[k] - Ps[ip].FL[k]) / T(2.0), lim_eps);
            Phis[k][i] = PhiR - PhiL;                                           // Phi*_{i+1/2}
        }
    }
    for (int i = 0; i < n; ++i) {
        int im = wrapi(i - 1, n);
        T gi = g ? g[i] : T(0.0);
        T S[5] = {T(0.0), us[0][i] * gi, T(0.0), T(0.0), us[1][i] * gi};
        for (int k = 0; k < 5; ++k)
            out[k][i] = u[k][i] - lam * (Phis[k][i] - Phis[k][im]) + kap * S[k];
    }
}

// Reverse pass of sweep_pencil, statement by statement.  Inputs: the sweep's INPUT pencil u,
// g, and ob = cotangent of the output.  Adds to ub (cotangent of u), gb (of g) and the three
// scalar cotangents.  Sub-gradient conventions R26.
void sweep_pencil_vjp(int n, const std::vector<double>* u, const double* g, double lam, double kap,
                      double gamma, double e_floor, double lim_eps,
                      const std::vector<double>* ob, std::vector<double>* ub, double* gb,
                      double& lam_b, double& kap_b, double& gamma_b) {
    // ---- recompute the forward intermediates (same statements as sweep_pencil<double>)
    std::vector<Prim<double>> P(n), Ps(n);
    std::vector<double> us[5], Phi[5], Phis[5];
    for (int k = 0; k < 5; ++k) { us[k].resize(n); Phi[k].resize(n); Phis[k].resize(n); }
    for (int i = 0; i < n; ++i) {
        double ui[5] = {u[0][i], u[1][i], u[2][i], u[3][i], u[4][i]};
        P[i] = prim(ui, gamma, e_floor);
    }
    for (int i = 0; i < n; ++i) {
        int ip = wrapi(i + 1, n);
        for (int k = 0; k < 5; ++k) Phi[k][i] = P[i].FR[k] - P[ip].FL[k];
    }
    for (int i = 0; i < n; ++i) {
        int im = wrapi(i - 1, n);
        double gi = g ? g[i] : 0.0;
        double S[5] = {0.0, u[0][i] * gi, 0.0, 0.0, u[1][i] * gi};
        for (int k = 0; k < 5; ++k)
            us[k][i] = u[k][i] - (lam / 2.0) * (Phi[k][i] - Phi[k][im]) + (kap / 2.0) * S[k];
    }
    for (int i = 0; i < n; ++i) {
        double ui[5] = {us[0][i], us[1][i], us[2][i], us[3][i], us[4][i]};
        Ps[i] = prim(ui, gamma, e_floor);
    }
    for (int i = 0; i < n; ++i) {
        int im = wrapi(i - 1, n), ip = wrapi(i + 1, n), ipp = wrapi(i + 2, n);
        for (int k = 0; k < 5; ++k) {
            double PhiR = Ps[i].FR[k] + limiter((Ps[i].FR[k] - Ps[im].FR[k]) / 2.0,
                                                (Ps[ip].FR[k] - Ps[i].FR[k]) / 2.0, lim_eps);
            double PhiL = Ps[ip].FL[k] - limiter((Ps[ip].FL[k] - Ps[i].FL[k]) / 2.0,
                                                 (Ps[ipp].FL[k] - Ps[ip].FL[k]) / 2.0, lim_eps);
            Phis[k][i] = PhiR - PhiL;
        }
    }
    // ---- reverse
    std::vector<double> usb[5], Phisb[5], Phib[5], FRsb[5], FLsb[5], FRb[5], FLb[5];
    for (int k = 0; k < 5; ++k) {
        usb[k].assign(n, 0.0); Phisb[k].assign(n, 0.0); Phib[k].assign(n, 0.0);
        FRsb[k].assign(n, 0.0); FLsb[k].assign(n, 0.0); FRb[k].assign(n, 0.0); FLb[k].assign(n, 0.0);
    }
    // out_i = u_i - lam (Phis_i - Phis_{i-1}) + kap S(us_i, g_i)
    for (int i = 0; i < n; ++i) {
        int im = wrapi(i - 1, n);
        double gi = g ? g[i] : 0.0;
        for (int k = 0; k < 5; ++k) {
            ub[k][i] += ob[k][i];
            lam_b += -ob[k][i] * (Phis[k][i] - Phis[k][im]);
            Phisb[k][i] += -lam * ob[k][i];
            Phisb[k][im] += lam * ob[k][i];
        }
        // S = (0, us_rho g, 0, 0, us_mn g)
        kap_b += ob[1][i] * us[0][i] * gi + ob[4][i] * us[1][i] * gi;
        usb[0][i] += kap * gi * ob[1][i];
        usb[1][i] += kap * gi * ob[4][i];
        if (gb) gb[i] += kap * (us[0][i] * ob[1][i] + us[1][i] * ob[4][i]);
    }
    // Phis_i = PhiR_i - PhiL_i
    for (int i = 0; i < n; ++i) {
        int im = wrapi(i - 1, n), ip = wrapi(i + 1, n), ipp = wrapi(i + 2, n);
        for (int k = 0; k < 5; ++k) {
            double PhiRb = Phisb[k][i], PhiLb = -Phisb[k][i];
            double da, db;
            // PhiR = FRs_i + phi(a,b), a = (FRs_i - FRs_im)/2, b = (FRs_ip - FRs_i)/2
            limiter_grad((Ps[i].FR[k] - Ps[im].FR[k]) / 2.0, (Ps[ip].FR[k] - Ps[i].FR[k]) / 2.0,
                         lim_eps, da, db);
            FRsb[k][i] += PhiRb;
            FRsb[k][i] += 0.5 * da * PhiRb;  FRsb[k][im] -= 0.5 * da * PhiRb;
            FRsb[k][ip] += 0.5 * db * PhiRb; FRsb[k][i] -= 0.5 * db * PhiRb;
            // PhiL = FLs_ip - phi(a,b), a = (FLs_ip - FLs_i)/2, b = (FLs_ipp - FLs_ip)/2
            limiter_grad((Ps[ip].FL[k] - Ps[i].FL[k]) / 2.0, (Ps[ipp].FL[k] - Ps[ip].FL[k]) / 2.0,
                         lim_eps, da, db);
            FLsb[k][ip] += PhiLb;
            FLsb[k][ip] -= 0.5 * da * PhiLb;  FLsb[k][i] += 0.5 * da * PhiLb;
            FLsb[k][ipp] -= 0.5 * db * PhiLb; FLsb[k][ip] += 0.5 * db * PhiLb;
        }
    }
    // (FRs_i, FLs_i) = prim(us_i)
    for (int i = 0; i < n; ++i) {
        double ui[5] = {us[0][i], us[1][i], us[2][i], us[3][i], us[4][i]};
        double a[5] = {FRsb[0][i], FRsb[1][i], FRsb[2][i], FRsb[3][i], FRsb[4][i]};
        double b[5] = {FLsb[0][i], FLsb[1][i], FLsb[2][i], FLsb[3][i], FLsb[4][i]};
        double t[5] = {0, 0, 0, 0, 0};
        prim_vjp(ui, gamma, e_floor, a, b, t, gamma_b);
        for (int k = 0; k < 5; ++k) usb[k][i] += t[k];
    }
    // us_i = u_i - (lam/2)(Phi_i - Phi_{i-1}) + (kap/2) S(u_i, g_i)
    for (int i = 0; i < n; ++i) {
        int im = wrapi(i - 1, n);
        double gi = g ? g[i] : 0.0;
        for (int k = 0; k < 5; ++k) {
            ub[k][i] += usb[k][i];
            lam_b += -0.5 * usb[k][i] * (Phi[k][i] - Phi[k][im]);
            Phib[k][i] += -0.5 * lam * usb[k][i];
            Phib[k][im] += 0.5 * lam * usb[k][i];
        }
        kap_b += 0.5 * (usb[1][i] * u[0][i] * gi + usb[4][i] * u[1][i] * gi);
        ub[0][i] += 0.5 * kap * gi * usb[1][i];
        ub[1][i] += 0.5 * kap * gi * usb[4][i];
        if (gb) gb[i] += 0.5 * kap * (u[0][i] * usb[1][i] + u[1][i] * usb[4][i]);
    }
    // Phi_i = FR_i - FL_{i+1}
    for (int i = 0; i < n; ++i) {
        int ip = wrapi(i + 1, n);
        for (int k = 0; k < 5; ++k) { FRb[k][i] += Phib[k][i]; FLb[k][ip] -= Phib[k][i]; }
    }
    // (FR_i, FL_i) = prim(u_i)
    for (int i = 0; i < n; ++i) {
        double ui[5] = {u[0][i], u[1][i], u[2][i], u[3][i], u[4][i]};
        double a[5] = {FRb[0][i], FRb[1][i], FRb[2][i], FRb[3][i], FRb[4][i]};
        double b[5] = {FLb[0][i], FLb[1][i], FLb[2][i], FLb[3][i], FLb[4][i]};
        double t[5] = {0, 0, 0, 0, 0};
        prim_vjp(ui, gamma, e_floor, a, b, t, gamma_b);
        for (int k = 0; k < 5; ++k) ub[k][i] += t[k];
    }
}

// ------------------------------------------------------------------ 3-D sweep -------
// Apply SWEEP_d to every pencil of a (nz, ny, nx) array stored C-order [z][y][x], x fastest.
// axis d: 0 = x, 1 = y, 2 = z.  gas = 5 fields (rho, m_x, m_y, m_z, eps), each nx*ny*nz.
// The normal momentum is field 1+d; transverse components keep cyclic order (d+1, d+2).
struct Dims { int nx, ny, nz; };

inline void pencil_geometry(Dims D, int d, int& n, long& stride, int& n1, long& s1, int& n2, long& s2) {
    long sx = 1, sy = D.nx, sz = (long)D.nx * D.ny;
    if (d == 0) { n = D.nx; stride = sx; n1 = D.ny; s1 = sy; n2 = D.nz; s2 = sz; }
    else if (d == 1) { n = D.ny; stride = sy; n1 = D.nx; s1 = sx; n2 = D.nz; s2 = sz; }
    else { n = D.nz; stride = sz; n1 = D.nx; s1 = sx; n2 = D.ny; s2 = sy; }
}

template <class T>
void sweep3d(Dims D, int d, const T* const gas_in[5], const T* g, T lam, T kap, T gamma,
             double e_floor, double lim_eps, T* const gas_out[5], double* cmax) {
    int n, n1, n2; long st, s1, s2;
    pencil_geometry(D, d, n, st, n1, s1, n2, s2);
    const int comp[5] = {0, 1 + d, 1 + (d + 1) % 3, 1 + (d + 2) % 3, 4};
    double cm_all = 0.0;
#pragma omp parallel for collapse(2) reduction(max : cm_all) schedule(static)
    for (int j2 = 0; j2 < n2; ++j2)
        for (int j1 = 0; j1 < n1; ++j1) {
            long base = j1 * s1 + j2 * s2;
            std::vector<T> u[5], out[5], gg(n);
            for (int k = 0; k < 5; ++k) {
                u[k].resize(n); out[k].resize(n);
                for (int i = 0; i < n; ++i) u[k][i] = gas_in[comp[k]][base + i * st];
            }
            if (g) for (int i = 0; i < n; ++i) gg[i] = g[base + i * st];
            double cm;
            sweep_pencil<T>(n, u, g ? gg.data() : nullptr, lam, kap, gamma, e_floor, lim_eps, out, &cm);
            cm_all = std::max(cm_all, cm);
            for (int k = 0; k < 5; ++k)
                for (int i = 0; i < n; ++i) gas_out[comp[k]][base + i * st] = out[k][i];
        }
    if (cmax) *cmax = cm_all;
}

// ub_in (5 fields) is OVERWRITTEN; gb (if not null) and the scalars are ACCUMULATED.
void sweep3d_vjp(Dims D, int d, const double* const gas_in[5], const double* g, double lam, double kap,
                 double gamma, double e_floor, double lim_eps, const double* const ob[5],
                 double* const ub_in[5], double* gb, double& lam_b, double& kap_b, double& gamma_b) {
    int n, n1, n2; long st, s1, s2;
    pencil_geometry(D, d, n, st, n1, s1, n2, s2);
    const int comp[5] = {0, 1 + d, 1 + (d + 1) % 3, 1 + (d + 2) % 3, 4};
    double lb = 0.0, kb = 0.0, gmb = 0.0;
#pragma omp parallel for collapse(2) reduction(+ : lb, kb, gmb) schedule(static)
    for (int j2 = 0; j2 < n2; ++j2)
        for (int j1 = 0; j1 < n1; ++j1) {
            long base = j1 * s1 + j2 * s2;
            std::vector<double> u[5], o[5], ub[5], gg(n), ggb(n, 0.0);
            for (int k = 0; k < 5; ++k) {
                u[k].resize(n); o[k].resize(n); ub[k].assign(n, 0.0);
                for (int i = 0; i < n; ++i) {
                    u[k][i] = gas_in[comp[k]][base + i * st];
                    o[k][i] = ob[comp[k]][base + i * st];
                }
            }
            if (g) for (int i = 0; i < n; ++i) gg[i] = g[base + i * st];
            double l1 = 0, k1 = 0, g1 = 0;
            sweep_pencil_vjp(n, u, g ? gg.data() : nullptr, lam, kap, gamma, e_floor, lim_eps, o, ub,
                             g ? ggb.data() : nullptr, l1, k1, g1);
            lb += l1; kb += k1; gmb += g1;
            for (int k = 0; k < 5; ++k)
                for (int i = 0; i < n; ++i) ub_in[comp[k]][base + i * st] = ub[k][i];
            if (g && gb) for (int i = 0; i < n; ++i) gb[base + i * st] += ggb[i];
        }
    lam_b += lb; kap_b += kb; gamma_b += gmb;
}

// ------------------------------------------------------------------------ FFT -------
// Own radix-2 decimation-in-time FFT (every config has N a power of two; no FFT library in the
// container).  X_k = sum_j x_j exp(sign * 2 pi i j k / n); unnormalised in both directions.
// Pinned against numpy.fft in tests.
template <class T>
struct Cx { T re, im; };

template <class T>
void fft1d(Cx<T>* a, int n, int sign) {
    for (int i = 1, j = 0; i < n; ++i) {               // bit reversal
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) std::swap(a[i], a[j]);
    }
    for (int len = 2; len <= n; len <<= 1) {
        for (int i = 0; i < n; i += len)
            for (int k = 0; k < len / 2; ++k) {
                double ang = sign * 2.0 * M_PI * k / len;
                double wr = std::cos(ang), wi = std::sin(ang);
                Cx<T> x = a[i + k], y = a[i + k + len / 2];
                Cx<T> t{y.re * T(wr) - y.im * T(wi), y.re * T(wi) + y.im * T(wr)};
                a[i + k] = Cx<T>{x.re + t.re, x.im + t.im};
                a[i + k + len / 2] = Cx<T>{x.re - t.re, x.im - t.im};
            }
    }
}

template <class T>
void fft3d(Cx<T>* a, int N, int sign) {
    long sx = 1, sy = N, sz = (long)N * N;
    long strides[3] = {sx, sy, sz};
    for (int ax = 0; ax < 3; ++ax) {
        long st = strides[ax], s1 = strides[(ax + 1) % 3], s2 = strides[(ax + 2) % 3];
#pragma omp parallel for collapse(2) schedule(static)
        for (int j2 = 0; j2 < N; ++j2)
            for (int j1 = 0; j1 < N; ++j1) {
                std::vector<Cx<T>> line(N);
                long base = j1 * s1 + j2 * s2;
                for (int i = 0; i < N; ++i) line[i] = a[base + i * st];
                fft1d(line.data(), N, sign);
                for (int i = 0; i < N; ++i) a[base + i * st] = line[i];
            }
    }
}

// ---------------------------------------------------------------- Poisson solve -----
// PAPER.md:71 ("forces are calculated via a potential formalism ... Fourier operators"),
// PAPER.md:83 (g = -grad phi).  Reading R12:  laplacian(phi') = A delta_tot,  g' = -grad phi',
//   g'^_d(k) = i k~_d A delta^(k) / k^2,  0 at k = 0,  k~_d = 0 on the axis-d Nyquist plane.
// k = (2 pi / L) n, n_d in (-N/2, N/2].  sign_mode = +1: forward operator G_d (d = 0,1,2 -> out[d]).
inline int kint(int j, int N) { return j <= N / 2 ? j : j - N; }

template <class T>
void poisson_force(int N, double L, T A, const T* delta, T* const gout[3]) {
    long n3 = (long)N * N * N;
    std::vector<Cx<T>> dh(n3);
    for (long c = 0; c < n3; ++c) dh[c] = Cx<T>{delta[c], T(0.0)};
    fft3d(dh.data(), N, -1);
    double kf = 2.0 * M_PI / L;
    for (int d = 0; d < 3; ++d) {
        std::vector<Cx<T>> gh(n3);
        for (int iz = 0; iz < N; ++iz)
            for (int iy = 0; iy < N; ++iy)
                for (int ix = 0; ix < N; ++ix) {
                    long c = ((long)iz * N + iy) * N + ix;
                    int nn[3] = {kint(ix, N), kint(iy, N), kint(iz, N)};
                    double kx = kf * nn[0], ky = kf * nn[1], kz = kf * nn[2];
                    double k2 = kx * kx + ky * ky + kz * kz;
                    double kd = (nn[d] == N / 2) ? 0.0 : kf * nn[d];
                    if (k2 == 0.0) { gh[c] = Cx<T>{T(0.0), T(0.0)}; continue; }
                    // i * kd * A / k2 * (re + i im) = (kd A / k2) * (-im + i re)
                    T s = T(kd / k2) * A;
                    gh[c] = Cx<T>{-(s * dh[c].im), s * dh[c].re};
                }
        fft3d(gh.data(), N, +1);
        for (long c = 0; c < n3; ++c) gout[d][c] = gh[c].re / T((double)n3);
    }
}

// transpose of poisson_force w.r.t. delta:  delta_b = sum_d G_d^T gb_d, written literally as
// (1/N^3) F^H conj(symbol) F gb_d, and A_b = sum_d <gb_d, g'_d> / A.
void poisson_force_vjp(int N, double L, double A, const double* const gb[3], double* delta_b) {
    long n3 = (long)N * N * N;
    std::vector<Cx<double>> acc(n3, Cx<double>{0.0, 0.0});
    double kf = 2.0 * M_PI / L;
    for (int d = 0; d < 3; ++d) {
        std::vector<Cx<double>> gh(n3);
        for (long c = 0; c < n3; ++c) gh[c] = Cx<double>{gb[d][c], 0.0};
        fft3d(gh.data(), N, -1);
        for (int iz = 0; iz < N; ++iz)
            for (int iy = 0; iy < N; ++iy)
                for (int ix = 0; ix < N; ++ix) {
                    long c = ((long)iz * N + iy) * N + ix;
                    int nn[3] = {kint(ix, N), kint(iy, N), kint(iz, N)};
                    double kx = kf * nn[0], ky = kf * nn[1], kz = kf * nn[2];
                    double k2 = kx * kx + ky * ky + kz * kz;
                    double kd = (nn[d] == N / 2) ? 0.0 : kf * nn[d];
                    if (k2 == 0.0) continue;
                    // conj(i s) * (re + i im) = -i s (re + i im) = s * (im - i re)
                    double s = kd * A / k2;
                    acc[c].re += s * gh[c].im;
                    acc[c].im += -s * gh[c].re;
                }
    }
    fft3d(acc.data(), N, +1);
    for (long c = 0; c < n3; ++c) delta_b[c] = acc[c].re / (double)n3;
}

// ---------------------------------------------------------------- cloud in cell -----
// PAPER.md:71 (particle-mesh), PAPER.md:244 (cloud-in-cell named).  Reading R13: mesh values
// live at cell centres (i + 1/2), so s = x - 1/2, i0 = floor(s), f = s - i0, i1 = i0 + 1, both
// wrapped mod N; weights (1-f | f) per axis.  The same (i0, f) serve deposit and gather.
template <class T>
struct Cic { int i0[3], i1[3]; T f[3]; };

template <class T>
inline Cic<T> cic_of(T x, T y, T z, int N) {
    Cic<T> C;
    T p[3] = {x, y, z};
    for (int d = 0; d < 3; ++d) {
        T s = p[d] - T(0.5);
        double fl = std::floor(val(s));
        C.f[d] = s - T(fl);
        int i0 = (int)fl;
        C.i0[d] = wrapi(i0, N);
        C.i1[d] = wrapi(i0 + 1, N);
    }
    return C;
}

template <class T>
void cic_deposit(int N, long np, const T* x, const T* y, const T* z, T mp, T* mesh) {
    for (long p = 0; p < np; ++p) {
        Cic<T> C = cic_of(x[p], y[p], z[p], N);
        for (int cz = 0; cz < 2; ++cz)
            for (int cy = 0; cy < 2; ++cy)
                for (int cx = 0; cx < 2; ++cx) {
                    T w = (cx ? C.f[0] : T(1.0) - C.f[0]) * (cy ? C.f[1] : T(1.0) - C.f[1]) *
                          (cz ? C.f[2] : T(1.0) - C.f[2]);
                    long c = ((long)(cz ? C.i1[2] : C.i0[2]) * N + (cy ? C.i1[1] : C.i0[1])) * N +
                             (cx ? C.i1[0] : C.i0[0]);
                    mesh[c] += mp * w;
                }
    }
}

template <class T>
inline T cic_gather_one(int N, const Cic<T>& C, const T* mesh) {
    T acc = T(0.0);
    for (int cz = 0; cz < 2; ++cz)
        for (int cy = 0; cy < 2; ++cy)
            for (int cx = 0; cx < 2; ++cx) {
                T w = (cx ? C.f[0] : T(1.0) - C.f[0]) * (cy ? C.f[1] : T(1.0) - C.f[1]) *
                      (cz ? C.f[2] : T(1.0) - C.f[2]);
                long c = ((long)(cz ? C.i1[2] : C.i0[2]) * N + (cy ? C.i1[1] : C.i0[1])) * N +
                         (cx ? C.i1[0] : C.i0[0]);
                acc += w * mesh[c];
            }
    return acc;
}

// d(gather)/d(position along axis d): the weight derivative is -1 (lower cell) / +1 (upper cell)
// along that axis; floor has zero derivative (R26).
inline double cic_gather_grad(int N, const Cic<double>& C, const double* mesh, int d) {
    double acc = 0.0;
    for (int cz = 0; cz < 2; ++cz)
        for (int cy = 0; cy < 2; ++cy)
            for (int cx = 0; cx < 2; ++cx) {
                int cc[3] = {cx, cy, cz};
                double w = 1.0;
                for (int e = 0; e < 3; ++e) {
                    if (e == d) w *= cc[e] ? 1.0 : -1.0;
                    else w *= cc[e] ? C.f[e] : 1.0 - C.f[e];
                }
                long c = ((long)(cz ? C.i1[2] : C.i0[2]) * N + (cy ? C.i1[1] : C.i0[1])) * N +
                         (cx ? C.i1[0] : C.i0[0]);
                acc += w * mesh[c];
            }
    return acc;
}

// ------------------------------------------------------------------ parameters ------
struct Params {
    int32_t N;            // grid cells per side
    int32_t n_part_side;  // particles per side (0 = no particles)
    double box;           // L, h^-1 Mpc (or code length in static mode)
    double gamma;
    double H0, Omega_m, Omega_b, Omega_L;
    int32_t static_mode;  // 1: a == 1 (config 1)
    int32_t gravity_on, hydro_on, gas_sources_gravity;
    double e_floor, lim_eps;
};

// Strang ordering ("XYZZYX, ZXYYXZ, YZXXZY"; reading R9): step n uses TABLE[n mod 6].
const int STRANG[6][3] = {{0, 1, 2}, {2, 1, 0}, {2, 0, 1}, {1, 0, 2}, {1, 2, 0}, {0, 2, 1}};

// Per-step scalars S0 (reading R15; Eq. 2-3 PAPER.md:61-63 give drift = int dt/a^2 and
// kick = int dt/a, evaluated by the midpoint rule at a_h = sqrt(a_i a_{i+1})).
struct Scalars { double dtau, kappa, K, A; };
inline Scalars step_scalars(const Params& P, double a_i, double a_next, double dt, double dt_prev) {
    Scalars S;
    if (P.static_mode) {
        S.dtau = dt; S.kappa = dt; S.K = 0.5 * (dt_prev + dt);
    } else {
        double ah = std::sqrt(a_i * a_next);
        S.dtau = dt / (ah * ah);
        S.kappa = dt / ah;
        S.K = (dt_prev + dt) / (2.0 * a_i);
    }
    S.A = 1.5 * P.Omega_m * P.H0 * P.H0;
    return S;
}

inline double f_baryon(const Params& P) { return P.Omega_m > 0 ? P.Omega_b / P.Omega_m : 0.0; }
inline long n_part(const Params& P) { return (long)P.n_part_side * P.n_part_side * P.n_part_side; }
inline double particle_mass(const Params& P) {
    long np = n_part(P);
    long n3 = (long)P.N * P.N * P.N;
    return np > 0 ? (1.0 - f_baryon(P)) * (double)n3 / (double)np : 0.0;
}
inline double rho_bar_src(const Params& P) {
    double m = 0.0;
    if (n_part(P) > 0) m += 1.0 - f_baryon(P);
    if (P.gas_sources_gravity) m += f_baryon(P);
    return m;
}

// ------------------------------------------------------------- the coupled step -----
// S1..S4 of SURVEY.md 8(c) (R16: one force field per step from the start-of-step state, used by
// both the particle kick and the three sweeps).  gas: 5*N^3, part: 6*np (x,y,z,wx,wy,wz),
// positions in grid units [0,N).  Scalars and gamma are of type T so the dual instantiation
// differentiates w.r.t. them too.  If sweep_inputs != nullptr the inputs of sweeps 2 and 3 are
// stored there (2 * 5 * N^3) for the reverse pass; gprime_out (3*N^3) likewise.
template <class T>
void step_core(const Params& P, T* gas, T* part, T dtau, T kappa, T K, T A, T gamma, int64_t step,
               double cmax[3], T* gprime_out, T* sweep_inputs) {
    const int N = P.N;
    const long n3 = (long)N * N * N;
    const long np = n_part(P);
    const double dx = P.box / N;
    std::vector<T> gp;       // g' (3 * n3)
    const bool grav = P.gravity_on != 0;
    if (grav) {
        // S1: Poisson source  delta_tot = rho_gas [if gas sources gravity] - rho_bar + CIC(particles)
        std::vector<T> delta(n3);
        const double rb = rho_bar_src(P);
        for (long c = 0; c < n3; ++c)
            delta[c] = (P.gas_sources_gravity ? gas[c] : T(0.0)) - T(rb);
        if (np > 0) cic_deposit<T>(N, np, part, part + np, part + 2 * np, T(particle_mass(P)), delta.data());
        // S2: g'
        gp.resize(3 * n3);
        T* gout[3] = {gp.data(), gp.data() + n3, gp.data() + 2 * n3};
        poisson_force<T>(N, P.box, A, delta.data(), gout);
        if (gprime_out) std::copy(gp.begin(), gp.end(), gprime_out);
    }
    // S3: particles -- gather, kick, drift, wrap (Eq. 2-3)
    if (np > 0) {
        T* x[3] = {part, part + np, part + 2 * np};
        T* w[3] = {part + 3 * np, part + 4 * np, part + 5 * np};
#pragma omp parallel for schedule(static)
        for (long p = 0; p < np; ++p) {
            if (grav) {
                Cic<T> C = cic_of(x[0][p], x[1][p], x[2][p], N);
                for (int d = 0; d < 3; ++d) w[d][p] += K * cic_gather_one<T>(N, C, gp.data() + d * n3);
            }
            for (int d = 0; d < 3; ++d) {
                T xn = x[d][p] + w[d][p] * dtau / T(dx);
                xn = xn - T((double)N * std::floor(val(xn) / N));
                if (val(xn) >= (double)N) xn = xn - T((double)N);
                x[d][p] = xn;
            }
        }
    }
    // S4: three sweeps in Strang order
    if (cmax) cmax[0] = cmax[1] = cmax[2] = 0.0;
    if (P.hydro_on) {
        std::vector<T> tmp(5 * n3);
        T lam = dtau / T(dx);
        Dims D{N, N, N};
        const int* order = STRANG[((step % 6) + 6) % 6];
        for (int s = 0; s < 3; ++s) {
            int d = order[s];
            if (sweep_inputs && s > 0) std::copy(gas, gas + 5 * n3, sweep_inputs + (long)(s - 1) * 5 * n3);
            const T* in[5]; T* out[5];
            for (int k = 0; k < 5; ++k) { in[k] = gas + k * n3; out[k] = tmp.data() + k * n3; }
            sweep3d<T>(D, d, in, grav ? gp.data() + d * n3 : nullptr, lam, kappa, gamma, P.e_floor,
                       P.lim_eps, out, cmax ? &cmax[s] : nullptr);
            std::copy(tmp.begin(), tmp.end(), gas);
        }
    }
}

// Reverse of step_core (SURVEY.md 8(c) "VJP structure").  gas_in / part_in: the step's INPUT state.
// cot_gas / cot_part: on entry cotangents of the step OUTPUT, on exit cotangents of the INPUT.
// dpar[5] += (dgamma, dDtau, dkappa, dK, dA).
void step_core_vjp(const Params& P, const double* gas_in, const double* part_in, double dtau,
                   double kappa, double K, double A, double gamma, int64_t step, double* cot_gas,
                   double* cot_part, double dpar[5]) {
    const int N = P.N;
    const long n3 = (long)N * N * N;
    const long np = n_part(P);
    const double dx = P.box / N;
    const bool grav = P.gravity_on != 0;
    // ---- recompute forward, keeping g' and the inputs of sweeps 2, 3
    std::vector<double> gas(gas_in, gas_in + 5 * n3), part(part_in, part_in + 6 * np);
    std::vector<double> gp(grav ? 3 * n3 : 0), sw(P.hydro_on ? 2 * 5 * n3 : 0);
    step_core<double>(P, gas.data(), part.data(), dtau, kappa, K, A, gamma, step, nullptr,
                      grav ? gp.data() : nullptr, P.hydro_on ? sw.data() : nullptr);
    std::vector<double> gpb(grav ? 3 * n3 : 0, 0.0);   // cotangent of g'
    double gamma_b = 0, dtau_b = 0, kappa_b = 0, K_b = 0, A_b = 0;
    // ---- S4 reversed
    if (P.hydro_on) {
        double lam = dtau / dx, lam_b = 0.0;
        Dims D{N, N, N};
        const int* order = STRANG[((step % 6) + 6) % 6];
        std::vector<double> tmp(5 * n3);
        for (int s = 2; s >= 0; --s) {
            int d = order[s];
            const double* src = (s == 0) ? gas_in : sw.data() + (long)(s - 1) * 5 * n3;
            const double* in[5]; const double* ob[5]; double* ub[5];
            for (int k = 0; k < 5; ++k) { in[k] = src + k * n3; ob[k] = cot_gas + k * n3; ub[k] = tmp.data() + k * n3; }
            sweep3d_vjp(D, d, in, grav ? gp.data() + d * n3 : nullptr, lam, kappa, gamma, P.e_floor,
                        P.lim_eps, ob, ub, grav ? gpb.data() + d * n3 : nullptr, lam_b, kappa_b, gamma_b);
            std::copy(tmp.begin(), tmp.end(), cot_gas);
        }
        dtau_b += lam_b / dx;
    }
    // ---- S3 reversed:  w' = w + K g_p(x);  x' = wrap(x + w' dtau/dx)
    std::vector<double> delta_b(grav ? n3 : 0, 0.0);
    if (np > 0) {
        const double* x[3] = {part_in, part_in + np, part_in + 2 * np};
        const double* w[3] = {part_in + 3 * np, part_in + 4 * np, part_in + 5 * np};
        double* xb[3] = {cot_part, cot_part + np, cot_part + 2 * np};
        double* wb[3] = {cot_part + 3 * np, cot_part + 4 * np, cot_part + 5 * np};
        for (long p = 0; p < np; ++p) {
            Cic<double> C = cic_of(x[0][p], x[1][p], x[2][p], N);
            double wtb[3], gpart[3] = {0, 0, 0};
            for (int d = 0; d < 3; ++d) {
                if (grav) gpart[d] = cic_gather_one<double>(N, C, gp.data() + d * n3);
                double wnew = w[d][p] + K * gpart[d];
                wtb[d] = wb[d][p] + (dtau / dx) * xb[d][p];      // total cotangent of w'
                dtau_b += xb[d][p] * wnew / dx;
                K_b += wtb[d] * gpart[d];
            }
            // x_b stays (wrap has unit derivative), w_b = wtb
            for (int d = 0; d < 3; ++d) wb[d][p] = wtb[d];
            if (grav) {
                // gather transposed: g'_b(cells) += W K wtb ; x_b += K sum_d wtb_d dg_p,d/dx
                for (int cz = 0; cz < 2; ++cz)
                    for (int cy = 0; cy < 2; ++cy)
                        for (int cx = 0; cx < 2; ++cx) {
                            double wt = (cx ? C.f[0] : 1.0 - C.f[0]) * (cy ? C.f[1] : 1.0 - C.f[1]) *
                                        (cz ? C.f[2] : 1.0 - C.f[2]);
                            long c = ((long)(cz ? C.i1[2] : C.i0[2]) * N + (cy ? C.i1[1] : C.i0[1])) * N +
                                     (cx ? C.i1[0] : C.i0[0]);
                            for (int d = 0; d < 3; ++d) gpb[d * n3 + c] += wt * K * wtb[d];
                        }
                for (int e = 0; e < 3; ++e) {
                    double acc = 0.0;
                    for (int d = 0; d < 3; ++d)
                        acc += K * wtb[d] * cic_gather_grad(N, C, gp.data() + d * n3, e);
                    xb[e][p] += acc;
                }
            }
        }
    }
    // ---- S2 reversed
    if (grav) {
        for (long c = 0; c < 3 * n3; ++c) A_b += gpb[c] * gp[c] / A;
        const double* gb3[3] = {gpb.data(), gpb.data() + n3, gpb.data() + 2 * n3};
        poisson_force_vjp(N, P.box, A, gb3, delta_b.data());
        // ---- S1 reversed
        if (P.gas_sources_gravity)
            for (long c = 0; c < n3; ++c) cot_gas[c] += delta_b[c];
        if (np > 0) {
            const double mp = particle_mass(P);
            const double* x[3] = {part_in, part_in + np, part_in + 2 * np};
            double* xb[3] = {cot_part, cot_part + np, cot_part + 2 * np};
#pragma omp parallel for schedule(static)
            for (long p = 0; p < np; ++p) {
                Cic<double> C = cic_of(x[0][p], x[1][p], x[2][p], N);
                for (int e = 0; e < 3; ++e) xb[e][p] += mp * cic_gather_grad(N, C, delta_b.data(), e);
            }
        }
    }
    dpar[0] += gamma_b; dpar[1] += dtau_b; dpar[2] += kappa_b; dpar[3] += K_b; dpar[4] += A_b;
}

}  // namespace

// =====================================================================================
// C interface (ctypes).  All arrays are host fp64, C-order [z][y][x]; gas = 5 fields
// (rho, m_x, m_y, m_z, eps) contiguous, part = 6 arrays (x, y, z, w_x, w_y, w_z) contiguous.
// =====================================================================================
extern "C" {

int orc_num_threads() {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

double orc_limiter(double a, double b, double eps) { return limiter<double>(a, b, eps); }

void orc_strang_order(int64_t step, int32_t out[3]) {
    const int* o = STRANG[((step % 6) + 6) % 6];
    out[0] = o[0]; out[1] = o[1]; out[2] = o[2];
}

// out[4] = (dtau, kappa, K, A)
void orc_step_scalars(const Params* P, double a_i, double a_next, double dt, double dt_prev, double out[4]) {
    Scalars S = step_scalars(*P, a_i, a_next, dt, dt_prev);
    out[0] = S.dtau; out[1] = S.kappa; out[2] = S.K; out[3] = S.A;
}

// Uniform-in-ln(a) schedule for a flat matter + Lambda cosmology: a_k = a0 exp(k r), dt_k = t(a_{k+1}) - t(a_k)
// with t(a) = int_0^a da' / (a' H(a')).  EdS closed form t = (2/3H0) a^{3/2}; otherwise Simpson quadrature.
void orc_schedule_lna(const Params* P, double a0, double a1, int n, double* a_out, double* dt_out) {
    double r = std::log(a1 / a0) / n;
    for (int k = 0; k <= n; ++k) a_out[k] = a0 * std::exp(k * r);
    a_out[n] = a1;
    for (int k = 0; k < n; ++k) {
        double lo = a_out[k], hi = a_out[k + 1];
        if (P->Omega_L == 0.0 && std::fabs(P->Omega_m - 1.0) < 1e-15) {
            dt_out[k] = (2.0 / (3.0 * P->H0)) * (std::pow(hi, 1.5) - std::pow(lo, 1.5));
        } else {
            const int M = 2000;   // Simpson in ln a
            double h = std::log(hi / lo) / M, acc = 0.0;
            for (int j = 0; j <= M; ++j) {
                double a = lo * std::exp(j * h);
                double Ok = 1.0 - P->Omega_m - P->Omega_L;
                double H = P->H0 * std::sqrt(P->Omega_m / (a * a * a) + Ok / (a * a) + P->Omega_L);
                double wgt = (j == 0 || j == M) ? 1.0 : (j % 2 ? 4.0 : 2.0);
                acc += wgt / H;
            }
            dt_out[k] = acc * h / 3.0;
        }
    }
}

// CIC cell index of fp32 positions, exactly as R13/R22: s = x - 0.5 (the fp32 value promoted to fp64,
// the subtraction is exact), i0 = floor(s) wrapped, i1 = i0 + 1 wrapped.
void orc_cell_index(const float* x, long n, int N, int32_t* i0, int32_t* i1) {
    for (long p = 0; p < n; ++p) {
        double s = (double)x[p] - 0.5;
        int f = (int)std::floor(s);
        i0[p] = wrapi(f, N);
        i1[p] = wrapi(f + 1, N);
    }
}

void orc_fft3(int N, const double* re_in, const double* im_in, int sign, double* re_out, double* im_out) {
    long n3 = (long)N * N * N;
    std::vector<Cx<double>> a(n3);
    for (long c = 0; c < n3; ++c) a[c] = Cx<double>{re_in[c], im_in ? im_in[c] : 0.0};
    fft3d(a.data(), N, sign);
    for (long c = 0; c < n3; ++c) { re_out[c] = a[c].re; im_out[c] = a[c].im; }
}

// general (nx, ny, nz) sweep; g may be null
void orc_sweep(int nx, int ny, int nz, int d, const double* gas_in, const double* g, double lam, double kap,
               double gamma, double e_floor, double lim_eps, double* gas_out, double* cmax) {
    long n3 = (long)nx * ny * nz;
    const double* in[5]; double* out[5];
    for (int k = 0; k < 5; ++k) { in[k] = gas_in + k * n3; out[k] = gas_out + k * n3; }
    sweep3d<double>(Dims{nx, ny, nz}, d, in, g, lam, kap, gamma, e_floor, lim_eps, out, cmax);
}

// JVP of the sweep: tangents of gas, g, and the scalars (dlam, dkap, dgamma)
void orc_sweep_jvp(int nx, int ny, int nz, int d, const double* gas_in, const double* g, double lam, double kap,
                   double gamma, double e_floor, double lim_eps, const double* dgas, const double* dg,
                   double dlam, double dkap, double dgamma, double* gas_out, double* dgas_out) {
    long n3 = (long)nx * ny * nz;
    std::vector<Dual> a(5 * n3), o(5 * n3), gg(g ? n3 : 0);
    for (long c = 0; c < 5 * n3; ++c) a[c] = Dual(gas_in[c], dgas ? dgas[c] : 0.0);
    if (g) for (long c = 0; c < n3; ++c) gg[c] = Dual(g[c], dg ? dg[c] : 0.0);
    const Dual* in[5]; Dual* out[5];
    for (int k = 0; k < 5; ++k) { in[k] = a.data() + k * n3; out[k] = o.data() + k * n3; }
    sweep3d<Dual>(Dims{nx, ny, nz}, d, in, g ? gg.data() : nullptr, Dual(lam, dlam), Dual(kap, dkap),
                  Dual(gamma, dgamma), e_floor, lim_eps, out, nullptr);
    for (long c = 0; c < 5 * n3; ++c) { gas_out[c] = o[c].v; dgas_out[c] = o[c].d; }
}

// VJP of the sweep: cot_in overwritten; gb accumulated; sc_b[3] += (lam_b, kap_b, gamma_b)
void orc_sweep_vjp(int nx, int ny, int nz, int d, const double* gas_in, const double* g, double lam, double kap,
                   double gamma, double e_floor, double lim_eps, const double* cot_out, double* cot_in,
                   double* gb, double sc_b[3]) {
    long n3 = (long)nx * ny * nz;
    const double* in[5]; const double* ob[5]; double* ub[5];
    for (int k = 0; k < 5; ++k) { in[k] = gas_in + k * n3; ob[k] = cot_out + k * n3; ub[k] = cot_in + k * n3; }
    sweep3d_vjp(Dims{nx, ny, nz}, d, in, g, lam, kap, gamma, e_floor, lim_eps, ob, ub, gb, sc_b[0], sc_b[1], sc_b[2]);
}

// mesh += mp * CIC(x)
void orc_deposit(int N, long np, const double* pos, double mp, double* mesh) {
    cic_deposit<double>(N, np, pos, pos + np, pos + 2 * np, mp, mesh);
}

// out[p] = CIC gather of mesh at particle p
void orc_gather(int N, long np, const double* pos, const double* mesh, double* out) {
    for (long p = 0; p < np; ++p) {
        Cic<double> C = cic_of(pos[p], pos[np + p], pos[2 * np + p], N);
        out[p] = cic_gather_one<double>(N, C, mesh);
    }
}

// gout: 3 * N^3
void orc_poisson(int N, double L, double A, const double* delta, double* gout) {
    long n3 = (long)N * N * N;
    double* g3[3] = {gout, gout + n3, gout + 2 * n3};
    poisson_force<double>(N, L, A, delta, g3);
}

void orc_poisson_vjp(int N, double L, double A, const double* gb, double* delta_b) {
    long n3 = (long)N * N * N;
    const double* g3[3] = {gb, gb + n3, gb + 2 * n3};
    poisson_force_vjp(N, L, A, g3, delta_b);
}

// One coupled step in place.  a, dt_prev, step are the state's scalars (updated: S5).
// cmax[3]: freezing-speed maxima of the three sweeps' inputs.  gprime_out (3 N^3) optional.
void orc_step(const Params* P, double* gas, double* part, double* a, double* dt_prev, int64_t* step,
              double dt, double a_next, double* cmax, double* gprime_out) {
    Scalars S = step_scalars(*P, *a, a_next, dt, *dt_prev);
    step_core<double>(*P, gas, part, S.dtau, S.kappa, S.K, S.A, P->gamma, *step, cmax, gprime_out, nullptr);
    *a = P->static_mode ? 1.0 : a_next;
    *dt_prev = dt;
    *step += 1;
}

// Same step with explicit scalars (used by the adjoint tests, which perturb the scalars).
void orc_step_explicit(const Params* P, double* gas, double* part, double dtau, double kappa, double K, double A,
                       double gamma, int64_t step) {
    step_core<double>(*P, gas, part, dtau, kappa, K, A, gamma, step, nullptr, nullptr, nullptr);
}

// JVP of the step with explicit scalars.  dscal[5] = tangents of (gamma, dtau, kappa, K, A).
void orc_step_jvp(const Params* P, const double* gas, const double* part, double dtau, double kappa, double K,
                  double A, double gamma, int64_t step, const double* dgas, const double* dpart,
                  const double* dscal, double* gas_out, double* part_out, double* dgas_out, double* dpart_out) {
    long n3 = (long)P->N * P->N * P->N, np = n_part(*P);
    std::vector<Dual> G(5 * n3), Q(6 * np);
    for (long c = 0; c < 5 * n3; ++c) G[c] = Dual(gas[c], dgas ? dgas[c] : 0.0);
    for (long c = 0; c < 6 * np; ++c) Q[c] = Dual(part[c], dpart ? dpart[c] : 0.0);
    step_core<Dual>(*P, G.data(), Q.data(), Dual(dtau, dscal[1]), Dual(kappa, dscal[2]), Dual(K, dscal[3]),
                    Dual(A, dscal[4]), Dual(gamma, dscal[0]), step, nullptr, nullptr, nullptr);
    for (long c = 0; c < 5 * n3; ++c) { gas_out[c] = G[c].v; dgas_out[c] = G[c].d; }
    for (long c = 0; c < 6 * np; ++c) { part_out[c] = Q[c].v; dpart_out[c] = Q[c].d; }
}

// VJP of the step with explicit scalars; cot_* in/out as in step_core_vjp; dpar[5] accumulated.
void orc_step_vjp_explicit(const Params* P, const double* gas_in, const double* part_in, double dtau, double kappa,
                           double K, double A, double gamma, int64_t step, double* cot_gas, double* cot_part,
                           double* dpar) {
    step_core_vjp(*P, gas_in, part_in, dtau, kappa, K, A, gamma, step, cot_gas, cot_part, dpar);
}

// VJP of the step as dh_step_vjp states it: (a_i, dt_prev, step) are the input state's scalars.
void orc_step_vjp(const Params* P, const double* gas_in, const double* part_in, double a_i, double dt_prev,
                  int64_t step, double dt, double a_next, double* cot_gas, double* cot_part, double* dpar) {
    Scalars S = step_scalars(*P, a_i, a_next, dt, dt_prev);
    step_core_vjp(*P, gas_in, part_in, S.dtau, S.kappa, S.K, S.A, P->gamma, step, cot_gas, cot_part, dpar);
}

// n steps forward from (gas, part, a0, dt_prev0 = 0, step0).  a_sched[k] = scale factor at the END of step k.
// cmax_out: 3 per step (optional).  states_out (optional): (n) input states, each 5 N^3 + 6 np doubles.
void orc_run(const Params* P, double* gas, double* part, double a0, int64_t step0, const double* a_sched,
             const double* dt_sched, int n, double* cmax_out, double* states_out) {
    long n3 = (long)P->N * P->N * P->N, np = n_part(*P);
    long ssz = 5 * n3 + 6 * np;
    double a = P->static_mode ? 1.0 : a0, dtp = 0.0;
    int64_t st = step0;
    for (int k = 0; k < n; ++k) {
        if (states_out) {
            std::copy(gas, gas + 5 * n3, states_out + k * ssz);
            std::copy(part, part + 6 * np, states_out + k * ssz + 5 * n3);
        }
        orc_step(P, gas, part, &a, &dtp, &st, dt_sched[k], a_sched[k], cmax_out ? cmax_out + 3 * k : nullptr, nullptr);
    }
}

// Reverse sweep over a run: forward storing every step's input, then step VJPs last to first.
// gas0/part0: initial state (not modified).  cot_gas/cot_part: cotangent of the FINAL state on entry,
// of the INITIAL state on exit.  dpar[5] accumulated over all steps.
void orc_run_vjp(const Params* P, const double* gas0, const double* part0, double a0, int64_t step0,
                 const double* a_sched, const double* dt_sched, int n, double* cot_gas, double* cot_part,
                 double* dpar) {
    long n3 = (long)P->N * P->N * P->N, np = n_part(*P);
    long ssz = 5 * n3 + 6 * np;
    std::vector<double> states((size_t)n * ssz), gas(gas0, gas0 + 5 * n3), part(part0, part0 + 6 * np);
    orc_run(P, gas.data(), part.data(), a0, step0, a_sched, dt_sched, n, nullptr, states.data());
    for (int k = n - 1; k >= 0; --k) {
        double a_i = P->static_mode ? 1.0 : (k == 0 ? a0 : a_sched[k - 1]);
        double dtp = k == 0 ? 0.0 : dt_sched[k - 1];
        orc_step_vjp(P, states.data() + k * ssz, states.data() + k * ssz + 5 * n3, a_i, dtp, step0 + k,
                     dt_sched[k], a_sched[k], cot_gas, cot_part, dpar);
    }
}

}  // extern "C"
