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

// The tables live outside the namespace with C linkage so inline PTX can name the symbol.
// TWO identical copies: the step loop addresses copy (step & 1), see TableBase below.
extern "C" {
__constant__ mgrhd::PlanckTables mgrhd_c_planck[2];
}

namespace mgrhd {

constexpr double kC15Pi4 = 0.15398973382026503;       // 15/pi^4

__device__ __forceinline__ double fast_rcp(double x);  // mgrhd_kernels.cuh

// Address (in the .const space) of one copy of the tables.  The caller derives `which` from the
// step counter of its loop: DFMA has no constant-bank operand form on sm_100, so a coefficient
// must be loaded into a (uniform) register either way, and when the table address is loop
// invariant ptxas hoists ALL ~100 coefficients of ALL branches ahead of the step loop, runs out
// of uniform registers and shuffles them through spills inside the loop (2-3 extra instructions
// per coefficient).  A base that changes with the step keeps each 16-byte load (two
// coefficients, one per Horner chain) next to its use.
struct TableBase { unsigned long long addr; };
__device__ __forceinline__ TableBase planck_table_base(int which) {
  unsigned long long a;
  asm("mov.u64 %0, mgrhd_c_planck;" : "=l"(a));
  TableBase t;
  t.addr = a + (unsigned long long)(which & 1) * sizeof(PlanckTables);
  return t;
}

template <int OFF>
__device__ __forceinline__ void ldc_pair(TableBase tb, double& a, double& b) {
  asm("ld.const.v2.f64 {%0, %1}, [%2+%3];" : "=d"(a), "=d"(b) : "l"(tb.addr), "n"(OFF));
}

// Two Horner chains sharing their coefficient loads: (sa, sb) <- (sa, sb) * t + table[N-1..0]
template <int BASE, int N>
__device__ __forceinline__ void horner_pair(TableBase tb, double t, double& sa, double& sb) {
  if constexpr (N > 0) {
    double ca, cb;
    ldc_pair<BASE + 16 * (N - 1)>(tb, ca, cb);
    sa = fma(sa, t, ca);
    sb = fma(sb, t, cb);
    horner_pair<BASE, N - 1>(tb, t, sa, sb);
  }
}

constexpr int kOffSp = 0;
constexpr int kOffMp = kOffSp + 16 * kSmallTerms;
constexpr int kOffL32 = kOffMp + 16 * kMidTerms;
constexpr int kOffL10 = kOffL32 + 16 * kLargeTerms;
constexpr int kOffMid = kOffL10 + 16 * kLargeTerms;

struct EdgeFn {
  double yz;   // Y(x) if small, else Z(x)
  double xi;   // Xi(x)
  bool small;  // which of the two yz holds
  int flops;   // algorithmic flop count of this evaluation (dead code unless counted)
};

// e^{-n x} series term n (1-based) folded into sum: sum <- sum*u + (l3 x^3 + l2 x^2 + l1 x + l0)
template <int N>
__device__ __forceinline__ void large_terms(TableBase tb, double x, double u, double& sum) {
  if constexpr (N > 0) {
    double c3, c2, c1, c0;
    ldc_pair<kOffL32 + 16 * (N - 1)>(tb, c3, c2);
    ldc_pair<kOffL10 + 16 * (N - 1)>(tb, c1, c0);
    const double pn = fma(fma(fma(c3, x, c2), x, c1), x, c0);
    sum = fma(sum, u, pn);
    large_terms<N - 1>(tb, x, u, sum);
  }
}

// x in [0, +inf].  x == 0 -> (Y=0, Xi=0); x == +inf or e^-x == 0 -> (Z=0, Xi=0).
__device__ __forceinline__ EdgeFn planck_edge(double x, TableBase tb) {
  EdgeFn r;
  if (x < kXS) {
    const double x2 = x * x;
    double sy, sx;
    ldc_pair<kOffSp + 16 * (kSmallTerms - 1)>(tb, sy, sx);
    horner_pair<kOffSp, kSmallTerms - 1>(tb, x2, sy, sx);
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
    double ms, mo;
    ldc_pair<kOffMid>(tb, ms, mo);
    const double t = fma(x, ms, mo);
    double sz, sx;
    ldc_pair<kOffMp + 16 * (kMidTerms - 1)>(tb, sz, sx);
    horner_pair<kOffMp, kMidTerms - 1>(tb, t, sz, sx);
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
  large_terms<kLargeTerms>(tb, x, u, sum);
  r.yz = sum * u;
  r.xi = kC15Pi4 * (x2 * x2) * (u * fast_rcp(1.0 - u));
  r.flops = kFlopEdgeLarge;
  return r;
}

// The same three branches for a CONVERGED warp: every branch that any lane needs is executed by
// all 32 lanes (a divergent branch costs the warp the same issue slots) and the result is kept by
// the lanes it belongs to.  Converged code lets the coefficient loads run on the uniform
// datapath, two coefficients per load, with no reconvergence bookkeeping.  `which` must be
// warp-uniform and change with the caller's loop counter (see TableBase above).
// x = NaN marks a lane without an edge: it matches no branch and gets (0, 0, large).
// One 16-byte load of a coefficient pair.
__device__ __forceinline__ double2 ld_pair(const Pair& p) { return *reinterpret_cast<const double2*>(&p); }

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

// Two edges at once (the same lane's edges of two consecutive steps): a branch needed by either
// edge of any lane is executed for BOTH edges by all lanes, so the four Horner chains interleave
// (DFMA latency is 8 cycles; two chains per warp leave the FP64 pipe half idle at 8 warps/SM) and
// each coefficient load feeds four DFMAs.
struct EdgeVal { double yz, xi; bool small; int flops; };

__device__ __forceinline__ void planck_edge_w2(double xa, double xb, int which, EdgeVal& A, EdgeVal& B) {
  const PlanckTables& tb = mgrhd_c_planck[which & 1];
  const unsigned FULL = 0xffffffffu;
  const bool aS = xa < kXS, aM = xa >= kXS && xa < kXL, aL = xa >= kXL;
  const bool bS = xb < kXS, bM = xb >= kXS && xb < kXL, bL = xb >= kXL;
  A.yz = 0.0; A.xi = 0.0; A.small = aS; A.flops = 0;
  B.yz = 0.0; B.xi = 0.0; B.small = bS; B.flops = 0;
  if (__any_sync(FULL, aS || bS)) {
    const double a2 = xa * xa, b2 = xb * xb;
    double2 cf = ld_pair(tb.sp[kSmallTerms - 1]);
    double ya = cf.x, za = cf.y, yb = cf.x, zb = cf.y;
#pragma unroll
    for (int n = kSmallTerms - 2; n >= 0; --n) {
      cf = ld_pair(tb.sp[n]);
      ya = fma(ya, a2, cf.x); za = fma(za, a2, cf.y);
      yb = fma(yb, b2, cf.x); zb = fma(zb, b2, cf.y);
    }
    const double ca3 = kC15Pi4 * (a2 * xa), cb3 = kC15Pi4 * (b2 * xb);
    // Y = C x^3 (1/3 - x/8 + x^2 sy),  Xi = C x^3 (1 - x/2 + x^2 sx)
    ya = ca3 * fma(a2, ya, fma(-0.125, xa, 1.0 / 3.0)); za = ca3 * fma(a2, za, fma(-0.5, xa, 1.0));
    yb = cb3 * fma(b2, yb, fma(-0.125, xb, 1.0 / 3.0)); zb = cb3 * fma(b2, zb, fma(-0.5, xb, 1.0));
    if (aS) { A.yz = ya; A.xi = za; A.flops = kFlopEdgeSmall; }
    if (bS) { B.yz = yb; B.xi = zb; B.flops = kFlopEdgeSmall; }
  }
  if (__any_sync(FULL, aM || bM)) {
    const double ta = fma(xa, tb.mid_s, tb.mid_o), tbb = fma(xb, tb.mid_s, tb.mid_o);
    double2 cf = ld_pair(tb.mp[kMidTerms - 1]);
    double za = cf.x, wa = cf.y, zb = cf.x, wb = cf.y;
#pragma unroll
    for (int n = kMidTerms - 2; n >= 0; --n) {
      cf = ld_pair(tb.mp[n]);
      za = fma(za, ta, cf.x); wa = fma(wa, ta, cf.y);
      zb = fma(zb, tbb, cf.x); wb = fma(wb, tbb, cf.y);
    }
    if (aM) { A.yz = za; A.xi = wa; A.flops = kFlopEdgeMid; }
    if (bM) { B.yz = zb; B.xi = wb; B.flops = kFlopEdgeMid; }
  }
  if (__any_sync(FULL, aL || bL)) {
    const double ua = exp(-xa), ub = exp(-xb);            // 0 on underflow and for x = +inf
    const double pa = aL && ua > 0.0 ? xa : 1.0;          // keeps inf * 0 out of the polynomials
    const double pb = bL && ub > 0.0 ? xb : 1.0;
    double sa = 0.0, sb = 0.0;
#pragma unroll
    for (int n = kLargeTerms - 1; n >= 0; --n) {
      const double2 c32 = ld_pair(tb.l32[n]), c10 = ld_pair(tb.l10[n]);
      sa = fma(sa, ua, fma(fma(fma(c32.x, pa, c32.y), pa, c10.x), pa, c10.y));
      sb = fma(sb, ub, fma(fma(fma(c32.x, pb, c32.y), pb, c10.x), pb, c10.y));
    }
    const double a2 = pa * pa, b2 = pb * pb;
    const double wa = kC15Pi4 * (a2 * a2) * (ua * fast_rcp(1.0 - ua));
    const double wb = kC15Pi4 * (b2 * b2) * (ub * fast_rcp(1.0 - ub));
    if (aL) { const bool l = ua > 0.0; A.yz = l ? sa * ua : 0.0; A.xi = l ? wa : 0.0; A.flops = l ? kFlopEdgeLarge : kFlopEdgeZero; }
    if (bL) { const bool l = ub > 0.0; B.yz = l ? sb * ub : 0.0; B.xi = l ? wb : 0.0; B.flops = l ? kFlopEdgeLarge : kFlopEdgeZero; }
  }
}

// Y(hi) - Y(lo) for two edges of one group (lo below hi).
__device__ __forceinline__ double planck_dY(const EdgeFn& lo, const EdgeFn& hi) {
  if (hi.small) return hi.yz - lo.yz;          // both small
  if (!lo.small) return lo.yz - hi.yz;         // both large: Z- - Z+
  return (1.0 - lo.yz) - hi.yz;                // straddling
}

}  // namespace mgrhd
