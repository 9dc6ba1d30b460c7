// mgrhd_planck.cuh -- device edge functions of the group Planck integral (Eq. 11
// applied to B_nu; "can be calculated analytically") in IEEE double.
//
//   Y(x)  = (15/pi^4) int_0^x t^3/(e^t-1) dt,   Z(x) = 1 - Y(x),
//   Xi(x) = (15/pi^4) x^4/(e^x-1)               (4 pi nu B_nu / c = a_R T^4 Xi(x)).
//
// Each edge returns ONE of Y (x < kXSplit, Maclaurin series in x^2) or Z (x >= kXSplit,
// sum_n e^{-nx}(x^3/n + 3x^2/n^2 + 6x/n^3 + 6/n^4)), so that a group difference never
// cancels in the Wien tail:  both small: Y+ - Y-;  both large: Z- - Z+;  straddling:
// 1 - Y- - Z+.
//
// Product code; independent of oracle/ (which sums in long double with a different split).
#pragma once
#include "mgrhd_params.h"

namespace mgrhd {

__constant__ PlanckTables c_planck;

constexpr double kXSplit = 1.5;                       // series switch
constexpr double kC15Pi4 = 0.15398973382026503;       // 15/pi^4

struct EdgeFn {
  double yz;   // Y(x) if small, else Z(x)
  double xi;   // Xi(x)
  bool small;  // which of the two yz holds
  int flops;   // algorithmic flop count of this evaluation (dead code unless counted)
};

// x in [0, +inf].  x == 0 -> (Y=0, Xi=0); x == +inf or e^-x == 0 -> (Z=0, Xi=0).
__device__ __forceinline__ EdgeFn planck_edge(double x) {
  EdgeFn r;
  if (x < kXSplit) {
    const double x2 = x * x;
    double sy = c_planck.y_c[kSmallTerms - 1];
    double sx = c_planck.xi_c[kSmallTerms - 1];
#pragma unroll
    for (int n = kSmallTerms - 2; n >= 0; --n) {
      sy = fma(sy, x2, c_planck.y_c[n]);
      sx = fma(sx, x2, c_planck.xi_c[n]);
    }
    const double x3 = x2 * x;
    // Y = C x^3 (1/3 - x/8 + x^2 sy),  Xi = C x^3 (1 - x/2 + x^2 sx)
    r.yz = kC15Pi4 * x3 * fma(x2, sy, fma(-0.125, x, 1.0 / 3.0));
    r.xi = kC15Pi4 * x3 * fma(x2, sx, fma(-0.5, x, 1.0));
    r.small = true;
    r.flops = kFlopEdgeSmall;
    return r;
  }
  r.small = false;
  const double u = exp(-x);
  if (!(u > 0.0)) {  // underflow or x = +inf
    r.yz = 0.0;
    r.xi = 0.0;
    r.flops = kFlopEdgeZero;
    return r;
  }
  const double x2 = x * x, x3 = x2 * x;
  const double c3 = x3, c2 = 3.0 * x2, c1 = 6.0 * x, c0 = 6.0;
  double un = u;     // u^n
  double sum = 0.0;
  int nt = 0;
  for (int n = 1; n <= kSeriesMax; ++n) {
    const double q = c_planck.inv_n[n];
    // x^3/n + 3x^2/n^2 + 6x/n^3 + 6/n^4  by Horner in 1/n
    const double pn = q * fma(q, fma(q, fma(q, c0, c1), c2), c3);
    const double term = un * pn;
    sum += term;
    ++nt;
    if (term <= 1e-18 * sum) break;
    un *= u;
  }
  r.yz = kC15Pi4 * sum;
  r.xi = kC15Pi4 * (x2 * x2) * (u / (1.0 - u));
  r.flops = kFlopEdgeLargeBase + kFlopEdgeTerm * nt;
  return r;
}

// Y(hi) - Y(lo) for two edges of one group (lo below hi).
__device__ __forceinline__ double planck_dY(const EdgeFn& lo, const EdgeFn& hi) {
  if (hi.small) return hi.yz - lo.yz;          // both small
  if (!lo.small) return lo.yz - hi.yz;         // both large: Z- - Z+
  return (1.0 - lo.yz) - hi.yz;                // straddling
}

}  // namespace mgrhd
