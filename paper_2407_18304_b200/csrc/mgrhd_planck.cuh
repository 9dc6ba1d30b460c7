// mgrhd_planck.cuh -- device edge functions of the group Planck integral (Eq. 11
// applied to B_nu; "can be calculated analytically") in IEEE double.
//
//   Y(x)  = (15/pi^4) int_0^x t^3/(e^t-1) dt,   Z(x) = 1 - Y(x),
//   Xi(x) = (15/pi^4) x^4/(e^x-1)               (4 pi nu B_nu / c = a_R T^4 Xi(x)).
//
// Each edge returns ONE of Y (x < kXS) or Z (x >= kXS), so that a group difference never
// cancels in the Wien tail:  both Y: Y+ - Y-;  both Z: Z- - Z+;  straddling: 1 - Y- - Z+.
// Three branches of BOUNDED cost (a warp evaluates one edge index at 32 temperatures, so the
// lanes of a warp usually share a branch; when they do not, the warp pays the sum):
//   x <  kXS        Maclaurin series in x^2, 12 even terms (truncation < 1e-19 relative);
//   kXS <= x < kXL  degree-23 polynomial fits of Z and Xi (Chebyshev interpolants generated
//                   in long double at init, abs. error < 1e-17 on functions of size 0.2-0.9);
//   x >= kXL        u = e^{-x}; Z = C sum_{n<=7} u^n (x^3/n + 3x^2/n^2 + 6x/n^3 + 6/n^4)
//                   (first dropped term < 3e-18 relative), Xi = C x^4 u/(1-u).
//
// Product code; independent of oracle/ (which sums both series in long double, split at x=1).
#pragma once
#include "mgrhd_params.h"

namespace mgrhd {

__constant__ PlanckTables c_planck;

constexpr double kC15Pi4 = 0.15398973382026503;       // 15/pi^4

__device__ __forceinline__ double fast_rcp(double x);  // mgrhd_kernels.cuh

struct EdgeFn {
  double yz;   // Y(x) if small, else Z(x)
  double xi;   // Xi(x)
  bool small;  // which of the two yz holds
  int flops;   // algorithmic flop count of this evaluation (dead code unless counted)
};

// x in [0, +inf].  x == 0 -> (Y=0, Xi=0); x == +inf or e^-x == 0 -> (Z=0, Xi=0).
__device__ __forceinline__ EdgeFn planck_edge(double x) {
  EdgeFn r;
  if (x < kXS) {
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
  if (x < kXL) {
    const double t = fma(x, c_planck.mid_s, c_planck.mid_o);
    double sz = c_planck.mz[kMidTerms - 1];
    double sx = c_planck.mx[kMidTerms - 1];
#pragma unroll
    for (int n = kMidTerms - 2; n >= 0; --n) {
      sz = fma(sz, t, c_planck.mz[n]);
      sx = fma(sx, t, c_planck.mx[n]);
    }
    r.yz = sz;
    r.xi = sx;
    r.flops = kFlopEdgeMid;
    return r;
  }
  const double u = exp(-x);
  if (!(u > 0.0)) {  // underflow or x = +inf
    r.yz = 0.0;
    r.xi = 0.0;
    r.flops = kFlopEdgeZero;
    return r;
  }
  const double x2 = x * x;
  double sum = 0.0;
#pragma unroll
  for (int n = kLargeTerms - 1; n >= 0; --n) {
    const double pn = fma(fma(fma(c_planck.l3[n], x, c_planck.l2[n]), x, c_planck.l1[n]), x, c_planck.l0[n]);
    sum = fma(sum, u, pn);
  }
  r.yz = sum * u;
  r.xi = kC15Pi4 * (x2 * x2) * (u * fast_rcp(1.0 - u));
  r.flops = kFlopEdgeLarge;
  return r;
}

// Y(hi) - Y(lo) for two edges of one group (lo below hi).
__device__ __forceinline__ double planck_dY(const EdgeFn& lo, const EdgeFn& hi) {
  if (hi.small) return hi.yz - lo.yz;          // both small
  if (!lo.small) return lo.yz - hi.yz;         // both large: Z- - Z+
  return (1.0 - lo.yz) - hi.yz;                // straddling
}

}  // namespace mgrhd
