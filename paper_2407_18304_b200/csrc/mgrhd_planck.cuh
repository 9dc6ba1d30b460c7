// mgrhd_planck.cuh -- device edge functions of the group Planck integral (Eq. 11
// applied to B_nu; "can be calculated analytically") in IEEE double.
//
//   Y(x)  = (15/pi^4) int_0^x t^3/(e^t-1) dt,   Z(x) = 1 - Y(x),
//   Xi(x) = (15/pi^4) x^4/(e^x-1)               (4 pi nu B_nu / c = a_R T^4 Xi(x)).
//
// Each edge returns ONE of Y (small x) or Z (large x), so that a group difference never
// cancels in the Wien tail:  both Y: Y+ - Y-;  both Z: Z- - Z+;  straddling: 1 - Y- - Z+.
//
// Two evaluations:
//  * planck_edge_t -- per-interval polynomial ROWS (58 intervals: [0, 0.5), eight per binade up to 64, x >= 64),
//    two degree-9 Horner chains whose coefficients each lane reads from its own row in shared memory:
//    ONE code path whatever the lanes' x (only e^-x for x >= 8 is a warp-wide branch).  Y below x = 1.
//    Used wherever the 10.2 KB of rows fit beside the kernel's state: every dispatched instantiation of the tuned
//    kernel and the general kernel.  Measured against the three-branch form at config 4: -12 % warp instructions,
//    -3 % time, 7 KB less code; at Nq = 64, where the rows cost a ninth warp, -4 %.
//  * planck_edge_w -- three warp-wide branches with uniform-register coefficients (below), Y below x = kXS;
//    for an instantiation whose group state fills shared memory (rows read from global memory instead were
//    15 % slower) and as the second form of the diagnostic entry point.
//
// planck_edge_w: three branches of BOUNDED cost:
//   x <  kXS        Maclaurin series in x^2, 12 even terms (truncation < 1e-19 relative);
//   kXS <= x < kXL  degree-23 polynomial fits of Z and Xi (Chebyshev interpolants generated
//                   in long double at init, abs. error < 1e-17 on functions of size 0.2-0.9);
//   x >= kXL        u = e^{-x}; Z = C sum_{n<=7} u^n (x^3/n + 3x^2/n^2 + 6x/n^3 + 6/n^4)
//                   (first dropped term < 3e-18 relative), Xi = C x^4 u/(1-u).
//
// Product code; independent of oracle/ (which sums both series in long double, split at x=1).
#pragma once
#include "mgrhd_params.h"

// The tables live outside the namespace with C linkage (one symbol, two identical copies; see
// planck_edge_w for why the second copy exists).
extern "C" {
__constant__ mgrhd::PlanckTables mgrhd_c_planck[2];
__device__ double mgrhd_g_rows[mgrhd::kRows * mgrhd::kRowStride];   // per-interval rows, copied to shared memory by the kernels
}

namespace mgrhd {

constexpr double kC15Pi4 = 0.15398973382026503;       // 15/pi^4

__device__ __forceinline__ double fast_rcp(double x);  // mgrhd_kernels.cuh

// One 16-byte load of a coefficient pair (one coefficient for each of two Horner chains).
__device__ __forceinline__ double2 ld_pair(const Pair& p) { return *reinterpret_cast<const double2*>(&p); }

// Edge functions for a CONVERGED warp: every branch that any lane needs is executed by all 32
// lanes (a divergent branch would cost the warp the same issue slots) and the result is kept by
// the lanes it belongs to.  Converged code lets the coefficient loads run on the uniform datapath
// with no reconvergence bookkeeping.  A warp evaluates neighbouring edge indices at 32/L
// temperatures, so its lanes usually share one or two branches.
//
// `which` must be warp-uniform, 0 at run time, and computed from the caller's loop counter in a
// way the compiler cannot fold (e.g. (i & 1) * P.zero): DFMA has no constant-bank operand form
// on sm_100, so each coefficient is loaded into a uniform register, and with a loop-invariant
// table address ptxas hoists all ~100 coefficients of all branches ahead of the caller's step
// loop, runs out of uniform registers and shuffles them through spills inside the loop (2-3
// extra instructions per coefficient).  Always reading copy 0 keeps the footprint in the
// constant cache at 1.1 KB.
//
// x in [0, +inf]; x == 0 -> (Y=0, Xi=0); x == +inf or e^-x == 0 -> (Z=0, Xi=0).
// x = NaN marks a lane without an edge: it matches no branch and gets (0, 0, large).
// flops: algorithmic flop count of the branch this lane's x falls in (dead code unless counted).
__device__ __forceinline__ void planck_edge_w(double x, int which, double& yz, double& xi, bool& small,
                                              int& flops) {
  const PlanckTables& tb = mgrhd_c_planck[which];
  const unsigned FULL = 0xffffffffu;
  const bool inS = x < kXS;
  const bool inM = x >= kXS && x < kXL;
  const bool inL = x >= kXL;
  yz = 0.0; xi = 0.0; small = inS; flops = 0;
  if (__any_sync(FULL, inS)) {
    const double x2 = x * x;
    double2 cf = ld_pair(tb.sp[kSmallTerms - 1]);
    double sy = cf.x, sx = cf.y;
#pragma unroll
    for (int n = kSmallTerms - 2; n >= 0; --n) {
      cf = ld_pair(tb.sp[n]);
      sy = fma(sy, x2, cf.x);
      sx = fma(sx, x2, cf.y);
    }
    const double cx3 = kC15Pi4 * (x2 * x);
    // Y = C x^3 (1/3 - x/8 + x^2 sy),  Xi = C x^3 (1 - x/2 + x^2 sx)
    const double y = cx3 * fma(x2, sy, fma(-0.125, x, 1.0 / 3.0));
    const double z = cx3 * fma(x2, sx, fma(-0.5, x, 1.0));
    if (inS) { yz = y; xi = z; flops = kFlopEdgeSmall; }
  }
  if (__any_sync(FULL, inM)) {
    const double t = fma(x, tb.mid_s, tb.mid_o);
    double2 cf = ld_pair(tb.mp[kMidTerms - 1]);
    double sz = cf.x, sx = cf.y;
#pragma unroll
    for (int n = kMidTerms - 2; n >= 0; --n) {
      cf = ld_pair(tb.mp[n]);
      sz = fma(sz, t, cf.x);
      sx = fma(sx, t, cf.y);
    }
    if (inM) { yz = sz; xi = sx; flops = kFlopEdgeMid; }
  }
  if (__any_sync(FULL, inL)) {
    const double u = exp(-x);            // 0 on underflow and for x = +inf
    const double xx = inL && u > 0.0 ? x : 1.0;   // keeps inf * 0 out of the polynomials
    double sum = 0.0;
#pragma unroll
    for (int n = kLargeTerms - 1; n >= 0; --n) {
      const double2 c32 = ld_pair(tb.l32[n]), c10 = ld_pair(tb.l10[n]);
      const double pn = fma(fma(fma(c32.x, xx, c32.y), xx, c10.x), xx, c10.y);
      sum = fma(sum, u, pn);
    }
    const double x2 = xx * xx;
    const double z = sum * u;
    const double w = kC15Pi4 * (x2 * x2) * (u * fast_rcp(1.0 - u));
    if (inL) {
      const bool live = u > 0.0;
      yz = live ? z : 0.0;
      xi = live ? w : 0.0;
      flops = live ? kFlopEdgeLarge : kFlopEdgeZero;
    }
  }
}

// One-branch edge functions: every lane reads the polynomial row of the interval its x falls in (16-byte pairs from
// shared memory, `rows` = a copy of mgrhd_g_rows) and runs two degree-9 Horner chains; only e^-x for x >= 8 is a
// warp-wide branch.  Same contract as planck_edge_w except that Y is returned below x = 1 (not kXS), Z from there
// on; NaN: no edge, (0, 0, large).  Accuracy: fit error < 1 ulp per row; Y = x^3 p(t) and Z = e^-x p(t) keep the
// relative accuracy in both tails.
__device__ __forceinline__ void planck_edge_t(double x, const double* rows, double& yz, double& xi, bool& small,
                                              int& flops) {
  const bool valid = x == x;
  const double xs = valid ? x : 2.0;
  int row = (__double2hiint(xs) >> 17) - (kRowKey0 - 1);
  row = row < 0 ? 0 : (row > kRows - 1 ? kRows - 1 : row);
  const double2* const r = reinterpret_cast<const double2*>(rows + row * kRowStride);
  const bool inY = xs < 1.0, inE = xs >= 8.0;
  double u = 1.0;
  if (__any_sync(0xffffffffu, inE)) u = exp(-xs);          // 0 on underflow and for x = +inf
  const bool live = !inE || u > 0.0;
  const double xx = live ? xs : 1.0;                        // keeps inf * 0 out of the polynomials
  const double2 cs = r[0];
  const double t = (xx - cs.x) * cs.y;
  double2 cf = r[kRowTerms];
  double sy = cf.x, sx = cf.y;
#pragma unroll
  for (int k = kRowTerms - 1; k >= 1; --k) {
    cf = r[k];
    sy = fma(sy, t, cf.x);
    sx = fma(sx, t, cf.y);
  }
  const double pref = inY ? xx * xx * xx : (inE ? u : 1.0);
  const bool keep = valid && live;
  yz = keep ? sy * pref : 0.0;
  xi = keep ? sx * pref : 0.0;
  small = valid && inY;
  flops = !valid ? 0 : (inY ? kFlopRowSmall : (!inE ? kFlopRowMid : (live ? kFlopRowLarge : kFlopEdgeZero)));
}

// The same for callers outside a step loop (table copy 0), compiled once and called: keeps a second
// copy of the three branches out of the hot kernel's instruction stream.
struct EdgeOut { double yz, xi; int small, flops; };
__device__ __noinline__ EdgeOut planck_edge_call(double x) {
  EdgeOut o;
  bool sm;
  planck_edge_w(x, 0, o.yz, o.xi, sm, o.flops);
  o.small = sm;
  return o;
}

// Edge functions of a cell's LOWEST edge, for a converged warp: the Rayleigh-Jeans branch inline
// (x_0 = h nu_0/(k_B T) is below kXS for any group structure that resolves the spectrum), anything
// else through planck_edge_call.  x = NaN: no edge, (0, 0, large).
__device__ __forceinline__ void planck_edge0(double x, double& yz, double& xi, bool& small, int& flops) {
  const PlanckTables& tb = mgrhd_c_planck[0];
  const bool inS = x < kXS;
  const double x2 = x * x;
  double2 cf = ld_pair(tb.sp[kSmallTerms - 1]);
  double sy = cf.x, sx = cf.y;
#pragma unroll
  for (int n = kSmallTerms - 2; n >= 0; --n) {
    cf = ld_pair(tb.sp[n]);
    sy = fma(sy, x2, cf.x);
    sx = fma(sx, x2, cf.y);
  }
  const double cx3 = kC15Pi4 * (x2 * x);
  yz = inS ? cx3 * fma(x2, sy, fma(-0.125, x, 1.0 / 3.0)) : 0.0;
  xi = inS ? cx3 * fma(x2, sx, fma(-0.5, x, 1.0)) : 0.0;
  small = inS;
  flops = inS ? kFlopEdgeSmall : 0;
  if (__any_sync(0xffffffffu, x >= kXS)) {
    const EdgeOut o = planck_edge_call(x);
    if (x >= kXS) { yz = o.yz; xi = o.xi; small = o.small != 0; flops = o.flops; }
  }
}

}  // namespace mgrhd
