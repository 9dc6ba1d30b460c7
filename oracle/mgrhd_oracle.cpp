// mgrhd_oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, single-threaded CPU oracle for the per-cell implicit
// matter-radiation source update of arXiv 2407.18304 (He, Wibking & Krumholz),
// written from /root/reference/PAPER.md only.  It shares no code, header,
// table or constant generator with the CUDA path under
// paper_2407_18304_b200/csrc/ and neither includes the other.  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
// may build, load or call it.
//
// What it computes: the paper's iteration, step by step in the paper's order
// (Eq. 37-52), with the dense (Nq+1)x(Nq+1) Jacobian of
// Eq. 48 assembled in full and solved by partial-pivot LU (no arrowhead
// shortcut on the update path).  Readings of garbled / silent passages are
// the S1..S18 readings of SURVEY.md section 8(c), restated in DESIGN.md.
//
// Arithmetic: IEEE double everywhere except inside the three Planck edge
// functions, which sum their defining series in long double so that the
// double results are correctly rounded to ~1 ulp.  Build with
//   g++ -O2 -std=c++17 -ffp-contract=off -shared -fPIC   (never -ffast-math).
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): adaptive quadrature of the
// Planck integrand, the printed T = 0.768032502191 of Eq. 56, the printed
// (3063.96, 101.248) of Eq. 63, Eq. 30 vs quadrature of Eq. 23, Eq. 26
// diffusion flux, conservation to round-off, the grey (Nq=1) limit of
// Eq. 5-6, the scalar monotone energy balance by bisection, a brute-force
// high-precision solve of the full (4+4Nq) system, arrowhead vs dense LU.
// Round 2 additions (each pinned in tests/test_oracle_next.py): the optional
// source term S_g; opacities evaluated at the
// trial temperature -- kappa_g (T/T_ref)^p and edge values
// tabulated in T with alpha from Eq. 20; the PPL free-slope
// spectrum fit of Appendix A.  For the free-slope fit the
// converged state is pinned (brute-force solve with the slopes recomputed at
// the root); from which iterate of E_g the slope alpha_E is taken during the
// iteration is a reading (S20) that only changes the iteration counts.  The
// 1-D transport at the end of this file follows a spatial scheme the paper
// does not give (reading S22): "parity unpinned" beyond the pins listed there.
// outer_mode 1 ("variant L", not in the paper) solves
// Eq. 51-52 implicitly in the velocity; its converged state is the same root
// of Eq. 37-40 and is pinned by the same brute-force solve.
//
// Notation (energy-density units, so 4*pi/c never appears):
//   x      = h nu / (k_B T)
//   Y(x)   = (15/pi^4) int_0^x t^3/(e^t-1) dt          in [0,1]
//   Z(x)   = 1 - Y(x)
//   Xi(x)  = (15/pi^4) x^4/(e^x-1)          (4 pi nu B_nu / c = a_R T^4 Xi)
//   Bt_g   = 4 pi B_g / c       = a_R T^4 [Y(x_g+) - Y(x_g-)]      (Eq. 11)
//   Db_g   = (4pi/c) Delta_g(nu B_nu)       = a_R T^4 [Xi(x_g+) - Xi(x_g-)]
//   D_g    = (4pi/c) Delta_g(nu chi0 B_nu)  = a_R T^4 [chi_g+ Xi(x_g+) - chi_g- Xi(x_g-)]

#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>

namespace {

const long double PI_L = 3.14159265358979323846264338327950288L;
const long double C15_PI4 = 15.0L / (PI_L * PI_L * PI_L * PI_L);

// Branch point between the Maclaurin series (x < XC) and the exponential
// series (x >= XC).  Any value in ~[0.5, 2] works; see S5.
const long double XC = 1.0L;

// Maclaurin coefficients b_k of t/(e^t-1) = sum_k b_k t^k  (b_k = B_k/k!),
// from the defining identity ((e^t-1)/t) * sum b_k t^k = 1:
//   sum_{j=0..k} b_j / (k-j+1)! = [k==0].
struct Maclaurin {
  static const int K = 48;
  long double b[K];
  Maclaurin() {
    long double invfact[K + 2];
    invfact[0] = 1.0L;
    for (int i = 1; i < K + 2; ++i) invfact[i] = invfact[i - 1] / (long double)i;
    b[0] = 1.0L;
    for (int k = 1; k < K; ++k) {
      long double s = 0.0L;
      for (int j = 0; j < k; ++j) s += b[j] * invfact[k - j + 1];
      b[k] = -s;  // divided by 1/1! = 1
    }
  }
};
const Maclaurin MAC;

// Y(x) for 0 <= x < XC:  t^3/(e^t-1) = sum_k b_k t^(k+2)  =>
//   int_0^x = sum_k b_k x^(k+3)/(k+3).                         (Eq. 11 with B_nu)
long double Y_small(long double x) {
  long double sum = 0.0L, xp = x * x * x;
  for (int k = 0; k < Maclaurin::K; ++k) {
    sum += MAC.b[k] * xp / (long double)(k + 3);
    xp *= x;
  }
  return C15_PI4 * sum;
}

// Z(x) = 1 - Y(x) for x >= XC:  1/(e^t-1) = sum_{n>=1} e^{-nt}  =>
//   int_x^inf t^3 e^{-nt} dt = e^{-nx} (x^3/n + 3x^2/n^2 + 6x/n^3 + 6/n^4).
long double Z_large(long double x) {
  if (std::isinf(x)) return 0.0L;
  long double sum = 0.0L;
  for (int n = 1; n <= 400; ++n) {
    long double nn = (long double)n;
    long double term = expl(-nn * x) *
        (x * x * x / nn + 3.0L * x * x / (nn * nn) + 6.0L * x / (nn * nn * nn) + 6.0L / (nn * nn * nn * nn));
    sum += term;
    if (term <= 1e-24L * sum) break;
  }
  return C15_PI4 * sum;
}

long double Xi_l(long double x) {
  if (x <= 0.0L || std::isinf(x)) return 0.0L;  // S6: Xi = 0 at edge 0 or inf
  return C15_PI4 * x * x * x * x / expm1l(x);
}

// Y(x+) - Y(x-) with no cancellation in the Wien tail (S5).
long double dY_l(long double xlo, long double xhi) {
  bool lo_small = xlo < XC, hi_small = xhi < XC;
  if (hi_small) return Y_small(xhi) - Y_small(xlo);           // both small
  if (!lo_small) return Z_large(xlo) - Z_large(xhi);          // both large
  return 1.0L - Y_small(xlo) - Z_large(xhi);                  // straddling
}

}  // namespace

extern "C" {

// ---- L1 special functions, exported so the tests can pin them ------------
double oracle_planck_Y(double x) {
  if (x <= 0.0) return 0.0;
  if (std::isinf(x)) return 1.0;
  return (double)((long double)x < XC ? Y_small(x) : 1.0L - Z_large(x));
}
double oracle_planck_Z(double x) {
  if (x <= 0.0) return 1.0;
  return (double)((long double)x < XC ? 1.0L - Y_small(x) : Z_large(x));
}
double oracle_planck_Xi(double x) { return (double)Xi_l(x); }
double oracle_planck_dY(double xlo, double xhi) { return (double)dY_l(xlo, xhi); }

}  // extern "C"

// ---------------------------------------------------------------------------
// L2: group-mean opacities, flux-mean opacity, closure
// ---------------------------------------------------------------------------
namespace {

// [ (r^p - 1)/p ] with the p -> 0 limit ln r.
double powint(double lnr, double p) {
  double z = p * lnr;
  if (z == 0.0) return lnr;
  return std::expm1(z) / p;
}

// minmod of Eq. A2: zero when the one-sided slopes differ in sign, else the one of smaller magnitude.
double minmod(double a, double b) {
  if (a * b <= 0.0) return 0.0;
  return std::fabs(a) < std::fabs(b) ? a : b;
}

}  // namespace

extern "C" {

// Appendix A, Eq. A1-A2: powerlaw indices alpha_{Q,g} of a radiation quantity from
// its group integrals Q[Nq].  Qbar_g = Q_g/(nu_g+ - nu_g-), nubar_g = sqrt(nu_g+ nu_g-),
// s_{g+1/2} = ln(Qbar_{g+1}/Qbar_g)/ln(nubar_{g+1}/nubar_g), alpha_g = minmod(s_{g-1/2}, s_{g+1/2});
// the two edge groups get -1.  Reading S21 (paper silent): a group whose own or whose neighbour's Q is
// not positive (the logarithm does not exist), or whose group structure has a zero or infinite edge,
// also gets -1, the fixed-slope value.
void oracle_free_slopes(int Nq, const double* edges, const double* Q, double* alphaQ) {
  for (int g = 0; g < Nq; ++g) alphaQ[g] = -1.0;
  for (int g = 1; g + 1 < Nq; ++g) {
    bool ok = true;
    double s[2];
    for (int k = 0; k < 2 && ok; ++k) {
      const int a = g - 1 + k, b = g + k;                    // the pair (a, b) = (g-1, g) then (g, g+1)
      const double wa = edges[a + 1] - edges[a], wb = edges[b + 1] - edges[b];
      if (!(Q[a] > 0.0) || !(Q[b] > 0.0) || !(edges[a] > 0.0) || !std::isfinite(edges[b + 1])) { ok = false; break; }
      const double na = std::sqrt(edges[a + 1] * edges[a]), nb = std::sqrt(edges[b + 1] * edges[b]);
      s[k] = std::log((Q[b] / wb) / (Q[a] / wa)) / std::log(nb / na);     // Eq. A1
    }
    if (ok) alphaQ[g] = minmod(s[0], s[1]);                                  // Eq. A2
  }
}

// Eq. 30 (reading S1): chi_{0Q,g} = chi_{0,g-} * [ (r^(aQ+1)-1)/(aQ+1) ]^-1
//                                              * [ (r^(ax+aQ+1)-1)/(ax+aQ+1) ].
// lnr = ln(nu_g+/nu_g-), a_chi = alpha_{chi0,g}, a_Q = alpha_{Q,g}.
double oracle_chi_mean(double chi_lo, double lnr, double a_chi, double a_Q) {
  if (a_chi == 0.0) return chi_lo;               // PC case
  return chi_lo * powint(lnr, a_chi + a_Q + 1.0) / powint(lnr, a_Q + 1.0);
}

// Eq. 27 with guard S8(i).  Bt, Db, D as in the header; aT4 = a_R T^4.
// Returns chi_F; *guard is set to 1 when the Wien-limit fallback was taken.
double oracle_chi_flux(double chiB, double chiE, double alpha, double chi_lo,
                       double Bt, double Db, double D, double aT4, int* guard) {
  double den = (4.0 / 3.0) * Bt - Db / 3.0;
  if (guard) *guard = 0;
  if (!(den >= 1e-280 * aT4) || !std::isfinite(den)) {
    if (guard) *guard = 1;
    return chi_lo;                               // analytic Wien limit of Eq. 27
  }
  double num = (chiB + chiE / 3.0) * Bt + (alpha * chiE * Bt - D) / 3.0;
  return num / den;
}

// Closure (reading S7): v^j P^{ji} for group energy E, flux F[3], velocity v[3].
// closure 0 = Levermore/M1, 1 = Eddington P = E/3 I.
void oracle_vP(int closure, double E, const double F[3], const double v[3], double c,
               double vP[3]) {
  double Fn = std::sqrt(F[0] * F[0] + F[1] * F[1] + F[2] * F[2]);
  if (closure == 1 || !(E > 0.0) || Fn == 0.0) {
    for (int i = 0; i < 3; ++i) vP[i] = E / 3.0 * v[i];
    return;
  }
  double f = Fn / (c * E);
  if (f > 1.0) f = 1.0;
  double chi = (3.0 + 4.0 * f * f) / (5.0 + 2.0 * std::sqrt(4.0 - 3.0 * f * f));
  double n[3] = {F[0] / Fn, F[1] / Fn, F[2] / Fn};
  double ndotv = n[0] * v[0] + n[1] * v[1] + n[2] * v[2];
  for (int i = 0; i < 3; ++i)
    vP[i] = E * (0.5 * (1.0 - chi) * v[i] + 0.5 * (3.0 * chi - 1.0) * n[i] * ndotv);
}

// The closure's pressure tensor P^{ji} itself (reading S7), for the implicit-in-v outer stage.
void oracle_P(int closure, double E, const double F[3], double c, double P[3][3]) {
  double e[3][3] = {{1, 0, 0}, {0, 1, 0}, {0, 0, 1}};
  for (int j = 0; j < 3; ++j) oracle_vP(closure, E, F, e[j], c, P[j]);     // row j = e_j . P
}

// Dense solve A x = b, partial-pivot LU, A row-major n x n (destroyed), b -> x.
// Returns 0, or -1 if a zero pivot is met.
int oracle_lu_solve(int n, double* A, double* b) {
  for (int k = 0; k < n; ++k) {
    int p = k;
    double best = std::fabs(A[k * n + k]);
    for (int i = k + 1; i < n; ++i)
      if (std::fabs(A[i * n + k]) > best) { best = std::fabs(A[i * n + k]); p = i; }
    if (best == 0.0) return -1;
    if (p != k) {
      for (int j = 0; j < n; ++j) { double t = A[k * n + j]; A[k * n + j] = A[p * n + j]; A[p * n + j] = t; }
      double t = b[k]; b[k] = b[p]; b[p] = t;
    }
    for (int i = k + 1; i < n; ++i) {
      double m = A[i * n + k] / A[k * n + k];
      if (m == 0.0) continue;
      for (int j = k; j < n; ++j) A[i * n + j] -= m * A[k * n + j];
      b[i] -= m * b[k];
    }
  }
  for (int i = n - 1; i >= 0; --i) {
    double s = b[i];
    for (int j = i + 1; j < n; ++j) s -= A[i * n + j] * b[j];
    b[i] = s / A[i * n + i];
  }
  return 0;
}

// The O(Nq) Gauss-Jordan elimination described at PAPER.md:440 for the
// arrowhead matrix of Eq. 48: J00, first row J0g[Nq], first column Jg0[Nq],
// diagonal Jgg[Nq]; rhs (-F_G, -F_R,g) in rhs[Nq+1] -> dx[Nq+1].
// Exported only so a test can check it against oracle_lu_solve.
void oracle_arrowhead_solve(int Nq, double J00, const double* J0g, const double* Jg0,
                            const double* Jgg, const double* rhs, double* dx) {
  double a = J00, r = rhs[0];
  for (int g = 0; g < Nq; ++g) {          // cancel first-row entries with rows 2..
    double m = J0g[g] / Jgg[g];
    a -= m * Jg0[g];
    r -= m * rhs[g + 1];
  }
  dx[0] = r / a;
  for (int g = 0; g < Nq; ++g) dx[g + 1] = (rhs[g + 1] - Jg0[g] * dx[0]) / Jgg[g];
}

}  // extern "C"

// ---------------------------------------------------------------------------
// L3: the per-cell implicit source update
// ---------------------------------------------------------------------------
extern "C" {

typedef struct {
  int Nq;
  const double* edges;      // [Nq+1] group edges nu_e (ascending, >= 0, last may be +inf)
  double a_rad, k_B, h_planck, mean_mass, gamma;
  const double* kappa_lo;   // [Nq] specific opacity at each group's LOWER edge (Eq. 19)
  const double* alpha;      // [Nq] in-group slope alpha_{chi0,g}  (0 => PC, Eq. 17)
  int closure;              // 0 Levermore/M1, 1 Eddington
  double newton_tol;        // epsilon of Eq. 49
  int newton_maxit;
  int outer_maxit;
  double outer_tol;         // 1e-13 of PAPER.md:465
  int outer_stop;           // 0 paper rule; 1 paper rule AND relative change of F_g, rho v (S10)
  double outer_rel_tol;     // 1e-12 (S10), used when outer_stop == 1
  // ---- round 2 ----
  int spectrum;             // 0 PPL fixed slope alpha_Q = -1; 1 free slope (Appendix A)
  int opacity_kind;         // 0 table (kappa_lo, alpha) independent of T
                            // 1 kappa_lo[g] (T/T_ref)^p_T, alpha as given
                            // 2 ln kappa tabulated at the Nq+1 EDGES on a uniform grid in ln T, alpha_g from the
                            //   two edge values of the group at the trial T (Eq. 20)
  double T_ref, p_T;        // kind 1
  int NT;                   // kind 2: temperatures in the table
  double lnT0, dlnT;        //         T_j = exp(lnT0 + j dlnT)
  const double* lnk_edge;   //         [Nq+1][NT] ln of the specific opacity at edge e, temperature j
  int outer_mode;           // 0: the paper's outer stage, velocity lagged in Eq. 51;
                            // 1: "variant L" of SURVEY 8(f) NEXT-4: v in Eq. 51 is the NEW velocity, so Eq. 51-52 are
                            //    one 3x3 linear system for v^(t+1) per outer trip (same fixed point; converges when the
                            //    radiation inertia q = (4/3) sum E_g/(rho c c_hat) is not small).  Not in the paper.
} oracle_model;

enum { ORACLE_HIST = 64 };
typedef struct {
  long long n_newton_unconverged;
  long long n_outer_unconverged;
  long long n_T_nonpositive_steps;
  long long n_chiF_guard;
  long long n_denominator_nonpositive;
  long long n_lu_singular;
  long long newton_evals_total;   // residual evaluations (O2-O6), summed over cells
  long long outer_trips_total;
  long long newton_hist[ORACLE_HIST];  // per-cell total Newton evaluations (clamped)
  long long outer_hist[ORACLE_HIST];   // per-cell outer trips (clamped)
} oracle_stats;

}  // extern "C"

namespace {

inline double norm3(const double a[3]) { return std::sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]); }

// One cell.  E[g], F[i][g] are the cell's group arrays; all updated in place.
// Specific opacity at edge e at temperature T for opacity_kind 2: linear interpolation of ln kappa in ln T
// between the two neighbouring table temperatures, the end values outside the table (reading S19).
double table_kappa(const oracle_model& m, int e, double T) {
  double u = (std::log(T) - m.lnT0) / m.dlnT;
  if (!(u > 0.0)) u = 0.0;
  if (u > (double)(m.NT - 1)) u = (double)(m.NT - 1);
  int j = (int)u;
  if (j > m.NT - 2) j = m.NT - 2;
  if (j < 0) j = 0;
  const double w = (m.NT > 1) ? u - (double)j : 0.0;
  const double* row = m.lnk_edge + (size_t)e * m.NT;
  const double lnk = (m.NT > 1) ? (1.0 - w) * row[j] + w * row[j + 1] : row[0];
  return std::exp(lnk);
}

// Ssrc: the cell's S_g [Nq], or null for S_g = 0.
void update_cell(const oracle_model& m, double dt, double c, double chat,
                 double rho, double kscale, double mom[3], double& Egas,
                 double* E, double* F0, double* F1, double* F2, const double* Ssrc, oracle_stats& st) {
  const int Nq = m.Nq;
  double* Fp[3] = {F0, F1, F2};
  std::vector<double> chi_lo(Nq), chi_hi(Nq), chiB(Nq), chiE(Nq), R(Nq, 0.0), Bt(Nq), Db(Nq), D(Nq),
      dBdT(Nq), chiF(Nq), W(Nq), Eg(Nq), FR(Nq), Enew(Nq), vF(Nq), xe(Nq + 1), Xi(Nq + 1), alpha(Nq), Sg(Nq, 0.0),
      alphaB(Nq, -1.0), alphaE(Nq, -1.0), Ecur(Nq), chi_edge(Nq + 1);
  if (Ssrc) Sg.assign(Ssrc, Ssrc + Nq);
  std::vector<double> Ft[3], Fk[3], Fnew[3];
  for (int i = 0; i < 3; ++i) { Ft[i].assign(Fp[i], Fp[i] + Nq); Fk[i] = Ft[i]; Fnew[i] = Ft[i]; }
  const std::vector<double> Et(E, E + Nq);
  const double Egas_t = Egas;
  const double mom_t[3] = {mom[0], mom[1], mom[2]};
  double mom_k[3] = {mom[0], mom[1], mom[2]}, mom_new[3] = {mom[0], mom[1], mom[2]};

  // O0/a3: opacities at the group edges (Eq. 19, 20) and group means (Eq. 30) at temperature T and, for the
  // free-slope spectrum, at the current iterate of the radiation energies.  For the T-independent table with
  // the fixed slope this is the same for every trial T (and is then what round 1 evaluated once per cell).
  auto opacities = [&](double T, const std::vector<double>& Bt_now, const std::vector<double>& E_now) {
    if (m.opacity_kind == 2)
      for (int e = 0; e <= Nq; ++e) chi_edge[e] = rho * kscale * table_kappa(m, e, T);
    if (m.spectrum == 1) {                                          // Appendix A, for B_g and for E_g alike
      oracle_free_slopes(Nq, m.edges, Bt_now.data(), alphaB.data());
      oracle_free_slopes(Nq, m.edges, E_now.data(), alphaE.data());
    }
    for (int g = 0; g < Nq; ++g) {
      double lnr = 0.0;
      if (m.opacity_kind == 2) {
        lnr = std::log(m.edges[g + 1] / m.edges[g]);
        chi_lo[g] = chi_edge[g];
        chi_hi[g] = chi_edge[g + 1];
        alpha[g] = std::log(chi_hi[g] / chi_lo[g]) / lnr;           // Eq. 20
      } else {
        alpha[g] = m.alpha[g];
        chi_lo[g] = rho * kscale * m.kappa_lo[g];
        if (m.opacity_kind == 1) chi_lo[g] *= std::pow(T / m.T_ref, m.p_T);
        if (alpha[g] != 0.0) {
          lnr = std::log(m.edges[g + 1] / m.edges[g]);
          chi_hi[g] = chi_lo[g] * std::exp(alpha[g] * lnr);         // Eq. 19 at nu_g+
        } else {
          chi_hi[g] = chi_lo[g];
        }
      }
      if (alpha[g] == 0.0) {
        chiB[g] = chiE[g] = chi_lo[g];                              // PC, Eq. 17
      } else {
        chiB[g] = oracle_chi_mean(chi_lo[g], lnr, alpha[g], alphaB[g]);   // Eq. 30; alpha_Q = -1 unless free slope
        chiE[g] = oracle_chi_mean(chi_lo[g], lnr, alpha[g], alphaE[g]);   // same method for both
      }
    }
  };
  double sumEt = 0.0, sumS = 0.0;
  for (int g = 0; g < Nq; ++g) { sumEt += Et[g]; sumS += Sg[g]; }
  const double Etot = Egas_t + (chat / c) * (sumEt + sumS);         // Eq. 50 as printed (S4)
  const double Cv = rho * m.k_B / ((m.gamma - 1.0) * m.mean_mass);  // S15

  double Egs = Egas_t;          // Newton iterate E_gas*
  double Egas_new = Egas_t;
  int newton_evals = 0, trips = 0;

  for (int k = 0; k < m.outer_maxit; ++k) {
    // O1: lagged velocity and fluxes
    double v[3] = {mom_k[0] / rho, mom_k[1] / rho, mom_k[2] / rho};
    double Ekin = (mom_k[0] * mom_k[0] + mom_k[1] * mom_k[1] + mom_k[2] * mom_k[2]) / (2.0 * rho);
    for (int g = 0; g < Nq; ++g) vF[g] = v[0] * Fk[0][g] + v[1] * Fk[1][g] + v[2] * Fk[2][g];
    if (!((Egs - Ekin) / Cv > 0.0)) { st.n_T_nonpositive_steps++; break; }  // invalid state: leave cell as is

    // inner Newton-Raphson on x = (E_gas, R_1..R_Nq)
    for (int it = 0;; ++it) {
      // O2: trial temperature and edge functions
      const double T = (Egs - Ekin) / Cv;
      const double aT4 = m.a_rad * T * T * T * T;
      for (int e = 0; e <= Nq; ++e) {
        double nu = m.edges[e];
        xe[e] = (nu == 0.0) ? 0.0 : (std::isinf(nu) ? nu : m.h_planck * nu / (m.k_B * T));
        Xi[e] = oracle_planck_Xi(xe[e]);
      }
      double sumR = 0.0, sumAbsFR = 0.0;
      // O3 (first half): group Planck integrals (Eq. 11); a3: opacities at this trial T; the free-slope fit
      // takes E_g at the current iterate, E_g^(t) + R_g + S_g (reading S20)
      for (int g = 0; g < Nq; ++g) {
        Bt[g] = aT4 * oracle_planck_dY(xe[g], xe[g + 1]);
        Ecur[g] = Et[g] + R[g] + Sg[g];
      }
      opacities(T, Bt, Ecur);
      for (int g = 0; g < Nq; ++g) {
        // O3: Doppler boundary terms (Eq. 18, 22)
        Db[g] = aT4 * (Xi[g + 1] - Xi[g]);
        D[g] = aT4 * (chi_hi[g] * Xi[g + 1] - chi_lo[g] * Xi[g]);
        dBdT[g] = (4.0 * Bt[g] - Db[g]) / T;
        // O4: flux-mean opacity (Eq. 27) and the work term of Eq. 21
        int guard = 0;
        chiF[g] = oracle_chi_flux(chiB[g], chiE[g], alpha[g], chi_lo[g], Bt[g], Db[g], D[g], aT4, &guard);
        if (guard && newton_evals == 0) st.n_chiF_guard++;
        if (!(1.0 + chat * chiF[g] * dt > 0.0)) {                  // S8(ii)
          if (newton_evals == 0) st.n_denominator_nonpositive++;
          chiF[g] = chiE[g];
        }
        W[g] = (1.0 + alpha[g]) * chiF[g] * vF[g] / c;
        // O5: Eq. 42 (reading S2) solved for E_g; residuals of Eq. 41
        Eg[g] = (chiB[g] / chiE[g]) * Bt[g] + W[g] / (c * chiE[g]) - R[g] / (chat * dt * chiE[g]);
        FR[g] = Eg[g] - Et[g] - (R[g] + Sg[g]);
        sumR += R[g];
        sumAbsFR += std::fabs(FR[g]);
      }
      const double FG = Egs - Egas_t + (c / chat) * sumR;
      newton_evals++;
      // O6: Eq. 49
      if (std::fabs(FG) / Etot < m.newton_tol && (c / chat) * sumAbsFR / Etot < m.newton_tol) break;
      if (it >= m.newton_maxit) { st.n_newton_unconverged++; break; }
      // O7: dense Jacobian of Eq. 44-48, solved by partial-pivot LU
      const int n = Nq + 1;
      std::vector<double> J((size_t)n * n, 0.0), dx(n);
      J[0] = 1.0;                                                    // Eq. 44
      dx[0] = -FG;
      for (int g = 0; g < Nq; ++g) {
        J[g + 1] = c / chat;                                         // Eq. 45
        J[(size_t)(g + 1) * n] = (chiB[g] / chiE[g]) * dBdT[g] / Cv; // Eq. 46 with d(chiB/chiE)/dT = 0
        J[(size_t)(g + 1) * n + g + 1] = -1.0 / (chat * dt * chiE[g]) - 1.0;  // Eq. 47
        dx[g + 1] = -FR[g];
      }
      if (oracle_lu_solve(n, J.data(), dx.data()) != 0) { st.n_lu_singular++; break; }
      // S9: keep T > 0 (halve the step, at most 10 times)
      double lam = 1.0;
      for (int h = 0; h < 10 && !((Egs + lam * dx[0] - Ekin) / Cv > 0.0); ++h) {
        lam *= 0.5;
        st.n_T_nonpositive_steps++;
      }
      Egs += lam * dx[0];
      for (int g = 0; g < Nq; ++g) R[g] += lam * dx[g + 1];
    }

    // O8: energy commit
    double sumR = 0.0;
    for (int g = 0; g < Nq; ++g) { Enew[g] = Et[g] + R[g] + Sg[g]; sumR += R[g]; }
    Egas_new = Egas_t - (c / chat) * sumR;

    // O9: flux update with the lagged velocity (Eq. 51); O10: gas momentum (Eq. 52)
    double dFsum[3] = {0.0, 0.0, 0.0};
    if (m.outer_mode == 1) {
      // variant L: Eq. 51 with the NEW velocity, F_g^new = a_g + B_g v^new, a_g = F_g^t/dn_g,
      // B_g = (c_hat dt/dn_g) [ (chi_B Bt - D/3) I + (1 + alpha) chi_E P_g ], dn_g = 1 + c_hat chi_F dt; inserted in Eq. 52:
      //   [rho I + (c c_hat)^-1 sum_g B_g] v^new = (rho v)^t - (c c_hat)^-1 sum_g (a_g - F_g^t)
      double M[9] = {rho, 0, 0, 0, rho, 0, 0, 0, rho}, rhs[3] = {mom_t[0], mom_t[1], mom_t[2]};
      std::vector<double> Bm((size_t)Nq * 9), av((size_t)Nq * 3);
      for (int g = 0; g < Nq; ++g) {
        double Fg[3] = {Fk[0][g], Fk[1][g], Fk[2][g]}, P[3][3];
        oracle_P(m.closure, Enew[g], Fg, c, P);
        const double dn = 1.0 + chat * chiF[g] * dt, A = chiB[g] * Bt[g] - D[g] / 3.0, w = (1.0 + alpha[g]) * chiE[g];
        for (int i = 0; i < 3; ++i) {
          av[(size_t)g * 3 + i] = Ft[i][g] / dn;
          rhs[i] -= (av[(size_t)g * 3 + i] - Ft[i][g]) / (c * chat);
          for (int j = 0; j < 3; ++j) {
            const double b = (chat * dt / dn) * ((i == j ? A : 0.0) + w * P[j][i]);
            Bm[(size_t)g * 9 + i * 3 + j] = b;
            M[i * 3 + j] += b / (c * chat);
          }
        }
      }
      if (oracle_lu_solve(3, M, rhs) != 0) { st.n_lu_singular++; break; }
      for (int g = 0; g < Nq; ++g)
        for (int i = 0; i < 3; ++i) {
          double f = av[(size_t)g * 3 + i];
          for (int j = 0; j < 3; ++j) f += Bm[(size_t)g * 9 + i * 3 + j] * rhs[j];
          Fnew[i][g] = f;
          dFsum[i] += f - Ft[i][g];
        }
    } else
    for (int g = 0; g < Nq; ++g) {
      double Fg[3] = {Fk[0][g], Fk[1][g], Fk[2][g]}, vP[3];
      oracle_vP(m.closure, Enew[g], Fg, v, c, vP);
      for (int i = 0; i < 3; ++i) {
        double src = v[i] * (chiB[g] * Bt[g] - D[g] / 3.0) + (1.0 + alpha[g]) * chiE[g] * vP[i];
        Fnew[i][g] = (Ft[i][g] + chat * dt * src) / (1.0 + chat * chiF[g] * dt);
        dFsum[i] += Fnew[i][g] - Ft[i][g];
      }
    }
    for (int i = 0; i < 3; ++i) mom_new[i] = mom_t[i] - dFsum[i] / (c * chat);   // Eq. 52 (variant L: = rho v^new up to rounding)
    trips++;

    // O11: outer convergence (reading S10)
    double vn[3] = {mom_new[0] / rho, mom_new[1] / rho, mom_new[2] / rho};
    double dW = 0.0, sumAbsR = 0.0;
    bool rel_ok = true;
    for (int g = 0; g < Nq; ++g) {
      double vFn = vn[0] * Fnew[0][g] + vn[1] * Fnew[1][g] + vn[2] * Fnew[2][g];
      double Wn = (1.0 + alpha[g]) * chiF[g] * vFn / c;
      dW += std::fabs(Wn - W[g]);
      sumAbsR += std::fabs(R[g]);
      if (m.outer_stop == 1) {
        double d[3] = {Fnew[0][g] - Fk[0][g], Fnew[1][g] - Fk[1][g], Fnew[2][g] - Fk[2][g]};
        double fn[3] = {Fnew[0][g], Fnew[1][g], Fnew[2][g]};
        if (!(norm3(d) <= m.outer_rel_tol * norm3(fn))) rel_ok = false;
      }
    }
    if (m.outer_stop == 1) {
      double d[3] = {mom_new[0] - mom_k[0], mom_new[1] - mom_k[1], mom_new[2] - mom_k[2]};
      if (!(norm3(d) <= m.outer_rel_tol * norm3(mom_new))) rel_ok = false;
    }
    const double delta = dW * (chat / c) * dt;
    const bool conv = (delta <= m.outer_tol * std::fmax(sumAbsR, Etot)) && rel_ok;
    if (conv) break;
    if (k == m.outer_maxit - 1) { st.n_outer_unconverged++; break; }
    for (int i = 0; i < 3; ++i) { mom_k[i] = mom_new[i]; Fk[i] = Fnew[i]; }
  }

  if (trips > 0) {
    for (int i = 0; i < 3; ++i) mom[i] = mom_new[i];
    Egas = Egas_new;  // total gas energy; E_int = Egas - |mom|^2/(2 rho)
    for (int g = 0; g < Nq; ++g) {
      E[g] = Enew[g];
      for (int i = 0; i < 3; ++i) Fp[i][g] = Fnew[i][g];
    }
  }
  st.newton_evals_total += newton_evals;
  st.outer_trips_total += trips;
  st.newton_hist[newton_evals < ORACLE_HIST ? newton_evals : ORACLE_HIST - 1]++;
  st.outer_hist[trips < ORACLE_HIST ? trips : ORACLE_HIST - 1]++;
}

}  // namespace

extern "C" {

// Host arrays, SoA, updated in place (rho, kappa_scale read-only):
//   rho[n], mom0/1/2[n], Egas[n], Erad[Nq][n], Frad0/1/2[Nq][n], kappa_scale[n] or NULL,
//   Srad[Nq][n] or NULL (the source term S_g of Eq. 41; read only).
// Returns 0, or a negative code for an argument error.
int oracle_source_update(const oracle_model* m, long long n, const double* rho,
                         double* mom0, double* mom1, double* mom2, double* Egas,
                         double* Erad, double* Frad0, double* Frad1, double* Frad2,
                         const double* kappa_scale, const double* Srad, double dt, double c, double chat,
                         oracle_stats* stats) {
  if (!m || m->Nq < 1 || !m->edges) return -1;
  if (m->opacity_kind < 0 || m->opacity_kind > 2 || m->spectrum < 0 || m->spectrum > 1) return -1;
  if (m->opacity_kind != 2 && (!m->kappa_lo || !m->alpha)) return -1;
  if (m->opacity_kind == 2 && (!m->lnk_edge || m->NT < 1 || (m->NT > 1 && !(m->dlnT > 0.0)))) return -1;
  if (m->opacity_kind == 1 && !(m->T_ref > 0.0)) return -2;
  if (!(dt > 0.0) || !(c > 0.0) || !(chat > 0.0) || chat > c) return -2;
  for (int g = 0; g < m->Nq; ++g) {
    if (!(m->edges[g + 1] > m->edges[g]) || m->edges[g] < 0.0) return -3;
    const bool open_group = m->edges[g] == 0.0 || std::isinf(m->edges[g + 1]);
    if (m->opacity_kind != 2 && m->alpha[g] != 0.0 && open_group) return -4;
    if (m->opacity_kind == 2 && open_group) return -4;      // Eq. 20 needs both edge values of every group
    if (m->opacity_kind != 2 && !(m->kappa_lo[g] > 0.0)) return -2;   // kappa = 0 makes Eq. 42 singular
  }
  oracle_stats st;
  std::memset(&st, 0, sizeof st);
  const int Nq = m->Nq;
  std::vector<double> E(Nq), F0(Nq), F1(Nq), F2(Nq), Sc(Nq);
  for (long long i = 0; i < n; ++i) {
    for (int g = 0; g < Nq; ++g) {
      if (Srad) Sc[g] = Srad[(size_t)g * n + i];
      E[g] = Erad[(size_t)g * n + i];
      F0[g] = Frad0[(size_t)g * n + i];
      F1[g] = Frad1[(size_t)g * n + i];
      F2[g] = Frad2[(size_t)g * n + i];
    }
    double mom[3] = {mom0[i], mom1[i], mom2[i]};
    double eg = Egas[i];
    update_cell(*m, dt, c, chat, rho[i], kappa_scale ? kappa_scale[i] : 1.0, mom, eg,
                E.data(), F0.data(), F1.data(), F2.data(), Srad ? Sc.data() : nullptr, st);
    mom0[i] = mom[0]; mom1[i] = mom[1]; mom2[i] = mom[2];
    Egas[i] = eg;
    for (int g = 0; g < Nq; ++g) {
      Erad[(size_t)g * n + i] = E[g];
      Frad0[(size_t)g * n + i] = F0[g];
      Frad1[(size_t)g * n + i] = F1[g];
      Frad2[(size_t)g * n + i] = F2[g];
    }
  }
  if (stats) *stats = st;
  return 0;
}

}  // extern "C"

// ---------------------------------------------------------------------------
// L4 (round 2): explicit radiation transport in 1-D and the two-stage
// IMEX step around the source update (Eq. 33-36).  TEST INFRASTRUCTURE.
//
// Eq. 34: dE_g/dt = -(c_hat/c) dF_g^x/dx,  dF_g^i/dt = -c c_hat dP_g^{xi}/dx  (1-D, x only), gas fields
// have no transport term.  The paper defers the spatial discretisation to "Paper II";
// the reading used by BOTH implementations (S22) is the plainest conservative one: piecewise
// constant states, local Lax-Friedrichs interface fluxes with the signal speed c_hat,
//   f_{i+1/2} = (f(u_i) + f(u_{i+1}))/2 - (c_hat/2)(u_{i+1} - u_i),
//   u = (E_g, F_g^x, F_g^y, F_g^z),  f(u) = ((c_hat/c) F^x, c c_hat P^{xx}, c c_hat P^{xy}, c c_hat P^{xz}),
// P_g from the closure of reading S7 (M1 or Eddington), periodic (bc = 0) or zero-gradient (bc = 1) ends.
// For a beam (|F| = cE along x) this is exact upwinding.  Parity unpinned beyond: conservation, the
// upwind closed form, uniform states, and the stage equations of Eq. 35-36 checked with the brute-force
// residual (tests/test_oracle_transport.py).
// ---------------------------------------------------------------------------
namespace {

// P^{x i} (i = x, y, z) of one group from (E, F): reading S7.
void pressure_x(int closure, double E, const double F[3], double c, double Px[3]) {
  double Fn = std::sqrt(F[0] * F[0] + F[1] * F[1] + F[2] * F[2]);
  if (closure == 1 || !(E > 0.0) || Fn == 0.0) {
    Px[0] = E / 3.0; Px[1] = 0.0; Px[2] = 0.0;
    return;
  }
  double f = Fn / (c * E);
  if (f > 1.0) f = 1.0;
  double chi = (3.0 + 4.0 * f * f) / (5.0 + 2.0 * std::sqrt(4.0 - 3.0 * f * f));
  double n[3] = {F[0] / Fn, F[1] / Fn, F[2] / Fn};
  for (int i = 0; i < 3; ++i) Px[i] = E * (0.5 * (3.0 * chi - 1.0) * n[0] * n[i]);
  Px[0] += E * 0.5 * (1.0 - chi);
}

}  // namespace

extern "C" {

// dst += wdt * T(src) for E_g and F_g of every group; nx cells along x (cell index fastest), spacing dx.
// src and dst may not alias.  Arrays as in oracle_source_update ([Nq][nx]).
int oracle_transport_add(int Nq, int closure, long long nx, double dx, double wdt, double c, double chat, int bc,
                         const double* sE, const double* sF0, const double* sF1, const double* sF2,
                         double* dE, double* dF0, double* dF1, double* dF2) {
  if (Nq < 1 || nx < 1 || !(dx > 0.0) || !(c > 0.0) || !(chat > 0.0) || bc < 0 || bc > 1) return -1;
  std::vector<double> flux((size_t)(nx + 1) * 4);   // interface i-1/2 at index i, i = 0..nx
  for (int g = 0; g < Nq; ++g) {
    const double* E = sE + (size_t)g * nx;
    const double* Fs[3] = {sF0 + (size_t)g * nx, sF1 + (size_t)g * nx, sF2 + (size_t)g * nx};
    auto cellidx = [&](long long i) -> long long {
      if (bc == 0) return (i % nx + nx) % nx;
      return i < 0 ? 0 : (i >= nx ? nx - 1 : i);
    };
    for (long long i = 0; i <= nx; ++i) {
      const long long a = cellidx(i - 1), b = cellidx(i);
      double Fa[3] = {Fs[0][a], Fs[1][a], Fs[2][a]}, Fb[3] = {Fs[0][b], Fs[1][b], Fs[2][b]}, Pa[3], Pb[3];
      pressure_x(closure, E[a], Fa, c, Pa);
      pressure_x(closure, E[b], Fb, c, Pb);
      double* f = &flux[(size_t)i * 4];
      f[0] = 0.5 * ((chat / c) * Fa[0] + (chat / c) * Fb[0]) - 0.5 * chat * (E[b] - E[a]);
      for (int k = 0; k < 3; ++k) f[1 + k] = 0.5 * (c * chat * Pa[k] + c * chat * Pb[k]) - 0.5 * chat * (Fb[k] - Fa[k]);
    }
    double* out[4] = {dE + (size_t)g * nx, dF0 + (size_t)g * nx, dF1 + (size_t)g * nx, dF2 + (size_t)g * nx};
    for (long long i = 0; i < nx; ++i)
      for (int k = 0; k < 4; ++k) out[k][i] += -(wdt / dx) * (flux[(size_t)(i + 1) * 4 + k] - flux[(size_t)i * 4 + k]);
  }
  return 0;
}

// One IMEX step of Eq. 35-36 in 1-D, in place (U^n -> U^(n+1)); Srad is not supported here (NULL).
//   stage 1: U* = U^n + dt T(U^n);  U^(n+1/2) = U* + dt S(U^(n+1/2))          (source update with theta = 1)
//   stage 2: U** = U^n + dt [T(U^n)/2 + T(U^(n+1/2))/2] + (dt/2) S(U^(n+1/2)) = (U^n + U^(n+1/2))/2 + (dt/2) T(U^(n+1/2))
//            (since dt S(U^(n+1/2)) = U^(n+1/2) - U* and dt T(U^n) = U* - U^n);  U^(n+1) = U** + (dt/2) S(U^(n+1))   (theta = 1/2)
int oracle_imex_step_1d(const oracle_model* m, long long nx, double dx, double dt, double c, double chat, int bc,
                        const double* rho, double* mom0, double* mom1, double* mom2, double* Egas, double* Erad,
                        double* Frad0, double* Frad1, double* Frad2, const double* kappa_scale, oracle_stats* stats) {
  if (!m) return -1;
  const size_t n = (size_t)nx, ng = (size_t)m->Nq * n;
  std::vector<double> w_m0(mom0, mom0 + n), w_m1(mom1, mom1 + n), w_m2(mom2, mom2 + n), w_eg(Egas, Egas + n),
      w_E(Erad, Erad + ng), w_F0(Frad0, Frad0 + ng), w_F1(Frad1, Frad1 + ng), w_F2(Frad2, Frad2 + ng);
  // stage 1
  int rc = oracle_transport_add(m->Nq, m->closure, nx, dx, dt, c, chat, bc, Erad, Frad0, Frad1, Frad2,
                                w_E.data(), w_F0.data(), w_F1.data(), w_F2.data());
  if (rc) return rc;
  oracle_stats s1, s2;
  rc = oracle_source_update(m, nx, rho, w_m0.data(), w_m1.data(), w_m2.data(), w_eg.data(), w_E.data(), w_F0.data(),
                            w_F1.data(), w_F2.data(), kappa_scale, nullptr, dt, c, chat, &s1);
  if (rc) return rc;
  // stage 2
  for (size_t i = 0; i < n; ++i) {
    mom0[i] = 0.5 * (mom0[i] + w_m0[i]); mom1[i] = 0.5 * (mom1[i] + w_m1[i]); mom2[i] = 0.5 * (mom2[i] + w_m2[i]);
    Egas[i] = 0.5 * (Egas[i] + w_eg[i]);
  }
  for (size_t i = 0; i < ng; ++i) {
    Erad[i] = 0.5 * (Erad[i] + w_E[i]);
    Frad0[i] = 0.5 * (Frad0[i] + w_F0[i]); Frad1[i] = 0.5 * (Frad1[i] + w_F1[i]); Frad2[i] = 0.5 * (Frad2[i] + w_F2[i]);
  }
  rc = oracle_transport_add(m->Nq, m->closure, nx, dx, 0.5 * dt, c, chat, bc, w_E.data(), w_F0.data(), w_F1.data(),
                            w_F2.data(), Erad, Frad0, Frad1, Frad2);
  if (rc) return rc;
  rc = oracle_source_update(m, nx, rho, mom0, mom1, mom2, Egas, Erad, Frad0, Frad1, Frad2, kappa_scale, nullptr,
                            0.5 * dt, c, chat, &s2);
  if (stats) {
    *stats = s2;
    stats->newton_evals_total += s1.newton_evals_total;
    stats->outer_trips_total += s1.outer_trips_total;
    stats->n_newton_unconverged += s1.n_newton_unconverged;
    stats->n_outer_unconverged += s1.n_outer_unconverged;
    stats->n_T_nonpositive_steps += s1.n_T_nonpositive_steps;
  }
  return rc;
}

}  // extern "C"
