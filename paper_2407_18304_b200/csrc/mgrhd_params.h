// mgrhd_params.h -- launch-time parameter block shared by the host API (mgrhd_api.cu) and
// the device kernels (mgrhd_kernels.cuh).  Passed BY VALUE as a __grid_constant__ kernel
// argument, so it lives in the constant bank: every table read below with a warp-uniform
// index is a uniform constant load, and several contexts can run concurrently on different
// streams without sharing a __constant__ symbol.
//
// Product code.  Shares nothing with oracle/.
#pragma once
#include "../../include/mgrhd.h"

namespace mgrhd {

constexpr int kMaxG = MGRHD_MAX_GROUPS;

// Device counters, one block of long long in global memory (see mgrhd_stats).
enum StatSlot {
  kStatCells = 0,
  kStatNewtonUnconv,
  kStatOuterUnconv,
  kStatTNonPos,
  kStatChiFGuard,
  kStatDenNonPos,
  kStatNewtonEvals,
  kStatOuterTrips,
  kStatFlops,                            // algorithmic FP64 flops (counting launches only)
  kStatNewtonHist,                       // MGRHD_HIST slots
  kStatOuterHist = kStatNewtonHist + MGRHD_HIST,
  kStatCount = kStatOuterHist + MGRHD_HIST
};

// Algorithmic FP64 flop counts of each piece of the update as written in mgrhd_kernels.cuh and
// mgrhd_planck.cuh (FMA = 2; add, mul, reciprocal/divide, sqrt = 1; exp = 30; comparisons, fabs,
// selects, shuffles = 0).  Derived line by line in DESIGN.md section 8; used only by the
// counting instantiations of the kernel (mgrhd_set_flop_counting), never in a timed run.
// A lane is charged for the ONE edge-function branch its x falls in, not for the branches it
// executes on behalf of other lanes of its warp.
constexpr int kFlopEdgeSmall = 59;    // x < kXS: x, x^2, two 12-term Horner chains in x^2, assembly
constexpr int kFlopEdgeMid = 95;      // kXS <= x < kXL: x, t, two degree-23 Horner chains
constexpr int kFlopEdgeLarge = 96;    // x >= kXL: x, exp, 7 terms of (3+1) FMA, Xi with one reciprocal
constexpr int kFlopEdgeZero = 32;     // x, exp that underflowed
constexpr int kFlopRowSmall = 43;     // planck_edge_t, x < 1: x (1), t (2), two degree-9 Horner chains (36), x^3 (2), x^3 p (2)
constexpr int kFlopRowMid = 39;       // planck_edge_t, 1 <= x < 8: x (1), t (2), two chains (36)
constexpr int kFlopRowLarge = 71;     // planck_edge_t, x >= 8: x (1), t (2), two chains (36), exp (30), e^-x p (2)
constexpr int kFlopGroupEval = 39;    // a2-a5 for one group at one trial T
constexpr int kFlopCellEval = 27;     // T, a_R T^4, beta, scales, v, F_G, Eq. 49, sums over the cell's lanes
constexpr int kFlopStepCell = 10;     // dx0, T > 0 check, E_gas update
constexpr int kFlopStepGroup = 4;     // R_g += lam da_g + (lam dx0) db_g
constexpr int kFlopOuterCell = 50;    // v, Eq. 52, commit, E_kin, outer tests, sums over the cell's lanes
constexpr int kFlopOuterGroup = 102;  // closure (46), Eq. 51 (23), relative-change test (14), sums (9), next v.F_g and dW (10)
constexpr int kFlopPowT = 64;         // opacity_kind 1: (T/T_ref)^p_T = exp(p ln(.)) (log 30, exp 30), chis, 1/chis
// the general kernel's model options (exp, log, expm1 = 30 each, like exp above)
constexpr int kFlopTabCell = 33;      // opacity_kind 2, per cell and evaluation: ln T, table position and weight
constexpr int kFlopTabEdge = 35;      // one edge opacity: two-point interpolation in ln T (4), exp, chi scale
constexpr int kFlopTabAlpha = 32;     // Eq. 20: ratio, log, division by ln r
constexpr int kFlopMeansVar = 6;      // means that change with the iterate: 3 chi_B + (1+alpha) chi_E (4), chi_B/chi_E (2)
constexpr int kFlopEq30Fixed = 34;    // Eq. 30 with alpha_Q = -1: z = alpha ln r, expm1, /alpha, /ln r, chi_lo x
constexpr int kFlopEq30Free = 66;     // Eq. 30 with a fitted slope: two brackets (mul, expm1, div each = 32), ratio, chi_lo x
constexpr int kFlopSlopeFit = 36;     // Eq. A1-A2 for one of B_g, E_g: Q/width, ratio, log, x 1/ln(nubar ratio), minmod (3)
constexpr int kFlopOuterGroupL = 126; // outer_mode 1: closure tensor (34), B_g (11), 6 matrix + 3 rhs sums (30), F_g^new (21), dF sums (6), test (14), next v.F_g and dW (10)
constexpr int kFlopOuterCellL = 107;  // outer_mode 1: kFlopOuterCell (50) + scaling the 9 sums (15), cofactors (18), determinant and reciprocal (6), v (18)
constexpr int kFlopCell = 16;         // load-time derivations
constexpr int kFlopCellGroup = 7;     // sum E_g, first v.F_g, E_g commit

struct Params {
  // ---- group structure and opacity table (set once by mgrhd_init) -------------------
  int Nq;
  int closure;        // 0 Levermore/M1, 1 Eddington
  int newton_maxit, outer_maxit, outer_stop;
  int zero;           // always 0: an opaque, loop-variant table offset (mgrhd_planck.cuh, planck_edge_w)
  double newton_tol, outer_tol, outer_rel_tol;
  double a_rad;
  double h_over_k;    // h / k_B : x_e = nu_e * h_over_k / T
  double cv_over_rho; // k_B / ((gamma-1) mean_mass)
  double nu[kMaxG + 1];     // group edges; nu[0] may be 0, nu[Nq] may be +inf
  double alpha[kMaxG];      // alpha_{chi0,g}
  double k_lo[kMaxG];       // kappa_lo[g]                       (chi_{g-} = rho*scale*k_lo)
  double k_hi[kMaxG];       // kappa_lo[g] * r_g^alpha_g         (chi_{g+}, Eq. 19 at nu_g+)
  double k_mean[kMaxG];     // kappa_lo[g] * (r^alpha-1)/(alpha ln r)   (Eq. 30 with alpha_Q=-1)
  double inv_k_mean[kMaxG]; // 1 / k_mean[g]
  double k_num[kMaxG];      // k_mean[g] * (4 + alpha_g)/3 : numerator factor of Eq. 27 with chi_B = chi_E
  double onepa[kMaxG];      // 1 + alpha_g (Eq. 21, 22)
  // ---- opacity_kind 1: chi scales with (T / T_ref)^p_T at every trial temperature ----
  double inv_T_ref, p_T;
  // ---- per call ------------------------------------------------------------------
  double dt, c, c_hat;
  long long ncells;   // cells in this launch
  long long stride;   // distance (in doubles) between consecutive groups in Erad/Frad
};

struct StatePtrs {
  const double* rho;
  double* mom[3];
  double* Egas;
  double* Erad;
  double* Frad[3];
  const double* kappa_scale;  // may be null
  const double* Srad;         // S_g [Nq][n], may be null
};

// Extra parameters of the general kernel (mgrhd_general.cuh): group geometry for Eq. 30 and Eq. A1-A2,
// the spectrum / opacity switches and the edge-opacity table of opacity_kind 2 (device memory).
struct GenParams {
  int spectrum;             // 0 fixed slope alpha_Q = -1, 1 free slope (Appendix A)
  int opacity_kind;         // 0, 1, 2 as in mgrhd_opacity_model
  int outer_mode;           // 0 lagged velocity in Eq. 51 (paper), 1 implicit in v ("variant L")
  int NT;
  double lnT0, inv_dlnT;
  const double* lnk_edge;   // device, [Nq+1][NT]
  double lnr[kMaxG];        // ln(nu_g+ / nu_g-); 0 for a group with an edge at 0 or +inf
  double width[kMaxG];      // nu_g+ - nu_g-  (Qbar_g = Q_g / width, Eq. A1)
  double inv_lnnb[kMaxG];   // 1 / ln(nubar_{g+1} / nubar_g), nubar = sqrt(nu_g+ nu_g-); 0 where Eq. A1 is undefined
};

// Tables of the Planck edge functions (mgrhd_planck.cuh), filled by the host once per device
// (mgrhd_api.cu: fill_planck_tables) and uploaded to __constant__ memory.
constexpr int kSmallTerms = 12;   // even Maclaurin terms, x < kXS
constexpr int kMidTerms = 24;     // monomial terms of the mid-range fits, kXS <= x < kXL
constexpr int kLargeTerms = 7;    // terms of the e^{-nx} series, x >= kXL
constexpr double kXS = 1.25;
constexpr double kXL = 5.5;
// Coefficients are stored in PAIRS (one 16-byte constant load feeds both Horner chains).
struct alignas(16) Pair { double a, b; };
struct alignas(16) PlanckTables {
  // t/(e^t-1) = 1 - t/2 + sum_{n>=1} b_{2n} t^(2n),  b_{2n} = B_{2n}/(2n)!
  //   sp[n-1] = { b_{2n}/(2n+3), b_{2n} } :  Y(x)  = C x^3 (1/3 - x/8 + sum sp[n-1].a x^(2n)),
  //                                          Xi(x) = C x^3 (1 - x/2 + sum sp[n-1].b x^(2n))
  Pair sp[kSmallTerms];
  // mid range: Z(x) = sum mp[k].a t^k, Xi(x) = sum mp[k].b t^k, t = mid_s * x + mid_o in [-1, 1]
  Pair mp[kMidTerms];
  // large x: Z(x) = C sum_{n=1..kLargeTerms} e^{-nx} (x^3/n + 3x^2/n^2 + 6x/n^3 + 6/n^4)
  Pair l32[kLargeTerms];      // { C/n, 3C/n^2 }
  Pair l10[kLargeTerms];      // { 6C/n^3, 6C/n^4 }
  double mid_s, mid_o;
};

// Per-interval polynomial rows of the edge functions (mgrhd_planck.cuh, planck_edge_t): row 0 is x in [0, 0.5), rows
// 1..56 the eight equal sub-intervals of each binade from [0.5, 1) to [32, 64) (the row index is read off the top bits
// of x), row 57 is x >= 64.  A row is kRowTerms + 1 pairs: {centre, 2/width}, then {a_k, b_k} for k = 0..kRowTerms-1:
//   x < 1:       Y  = x^3 sum a_k t^k,     Xi = x^3 sum b_k t^k      (15/pi^4 folded in)
//   1 <= x < 8:  Z  = sum a_k t^k,         Xi = sum b_k t^k
//   x >= 8:      Z  = e^-x sum a_k t^k,    Xi = e^-x sum b_k t^k,     t = (x - centre) 2/width  (row 57: t = x)
constexpr int kRows = 58;
constexpr int kRowTerms = 10;                      // degree 9: fit error below 1 ulp on every row
constexpr int kRowStride = 2 * (kRowTerms + 1);    // doubles; 176 B puts eight neighbouring rows on distinct banks
constexpr int kRowKey0 = 1022 * 8;                 // (high word >> 17) of 0.5

}  // namespace mgrhd
