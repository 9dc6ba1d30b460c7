// mgrhd_transport.cuh -- explicit radiation transport T(U) of Eq. 34 in 1-D and the
// element-wise helper of the two-stage IMEX step (Eq. 35-36).  SURVEY 8(f) NEXT-3.
//
//   dE_g/dt = -(c_hat/c) dF_g^x/dx,   dF_g^i/dt = -c c_hat dP_g^{xi}/dx,   gas fields: no transport term.
//
// The paper defers the spatial discretisation to Paper II; the reading used here and in the oracle
// (S22) is piecewise-constant states with local Lax-Friedrichs interface fluxes at the signal
// speed c_hat:  f_{i+1/2} = (f(u_i) + f(u_{i+1}))/2 - (c_hat/2)(u_{i+1} - u_i),  u = (E, F^x, F^y, F^z),
// f(u) = ((c_hat/c) F^x, c c_hat P^xx, c c_hat P^xy, c c_hat P^xz), P from the closure of reading S7.
//
// HBM-bound: per cell-group the kernel reads u of the source state (4 doubles; the two halo cells of a tile
// are re-read from L2), reads and writes u of the destination (4 + 4): 96 algorithmic bytes.  One thread per
// (group, cell): f(u_i) is formed once per cell (one closure: two sqrt, two divisions), staged with u_i in
// shared memory, and each interior thread of the tile combines its interfaces.  Tiles overlap by one thread's
// cells on each side, so 254/256 of the threads produce output; the cell index is the fastest in memory, so every
// load and store of a warp is one contiguous run.  The destination's old values are loaded up front, so a
// thread has eight loads in flight, and with an even nx a thread owns two neighbouring cells and moves them with
// 16-byte accesses (measured at 256^3 x 32: 4.1 TB/s for the first version with the read-modify-write after the
// barrier and four divisions per closure; 5.4 TB/s with the loads up front; 5.75 TB/s = 0.88 of the measured
// HBM peak with two cells per thread).
//
// Product code; shares nothing with oracle/.
#pragma once
#include "mgrhd_params.h"

namespace mgrhd {

constexpr int kTransportTile = 256;

// P^{x i} c c_hat and (c_hat/c) F^x of one cell-group: the flux vector f(u).
__device__ __forceinline__ void transport_flux(int closure, double E, double F0, double F1, double F2, double c,
                                               double chat, double (&f)[4]) {
  const double Fn = sqrt(F0 * F0 + F1 * F1 + F2 * F2);
  double Pxx = E / 3.0, Pxy = 0.0, Pxz = 0.0;
  if (!(closure == 1 || !(E > 0.0) || Fn == 0.0)) {
    double ff = Fn / (c * E);
    if (ff > 1.0) ff = 1.0;
    // Levermore 1984: chi = (3 + 4 f^2)/(5 + 2 s), s = sqrt(4 - 3 f^2), equals (5 - 2 s)/3, so
    // (1 - chi)/2 = (s - 1)/3 and (3 chi - 1)/2 = 2 - s: no division
    const double sq = sqrt(4.0 - 3.0 * ff * ff);
    const double rF = 1.0 / Fn;
    const double n0 = F0 * rF, n1 = F1 * rF, n2 = F2 * rF;
    const double an = E * (2.0 - sq);
    Pxx = an * n0 * n0 + E * ((sq - 1.0) * (1.0 / 3.0));
    Pxy = an * n0 * n1;
    Pxz = an * n0 * n2;
  }
  f[0] = (chat / c) * F0;
  f[1] = c * chat * Pxx;
  f[2] = c * chat * Pxy;
  f[3] = c * chat * Pxz;
}

// dst(E_g, F_g) += wdt * T(src) for nx cells; V cells per thread (V = 2: 16-byte loads and stores, needs an even
// nx so that every group row starts on a 16-byte boundary); grid = (ceil(nx / (V (tile - 2))), Nq), block = tile
// threads.  bc: 0 periodic, 1 zero-gradient.  src and dst must not alias.
template <int V>
__global__ void __launch_bounds__(kTransportTile)
transport_add_kernel(const __grid_constant__ StatePtrs src, const __grid_constant__ StatePtrs dst, int closure,
                     long long nx, long long stride_src, long long stride_dst, double wdt_over_dx, double c,
                     double chat, int bc) {
  constexpr int NC = V * kTransportTile;            // cells staged per tile (V halo cells on each side)
  __shared__ __align__(16) double s_u[4][NC];
  __shared__ __align__(16) double s_f[4][NC];
  const int t = threadIdx.x;
  const long long g = blockIdx.y;
  const long long i0 = (long long)blockIdx.x * (NC - 2 * V) + (long long)V * t - V;   // first of this thread's V cells
  const double* const in[4] = {src.Erad, src.Frad[0], src.Frad[1], src.Frad[2]};
  double* const out[4] = {dst.Erad, dst.Frad[0], dst.Frad[1], dst.Frad[2]};
  const bool writer = t >= 1 && t <= kTransportTile - 2 && i0 < nx;
  const bool in_range = i0 <= nx;                   // (cells beyond nx + V - 1 are never needed)
  double u[4][V], d[4][V];
#pragma unroll
  for (int k = 0; k < 4; ++k)
#pragma unroll
    for (int m = 0; m < V; ++m) { u[k][m] = 0.0; d[k][m] = 0.0; }
  // the destination's old values first: in flight together with the source loads
  const bool full = V == 2 && i0 >= 0 && i0 + 1 < nx;      // both cells inside the row: one aligned 16-byte access
  if (writer) {
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      if (V == 2 && full) {
        const double2 q = *reinterpret_cast<const double2*>(out[k] + g * stride_dst + i0);
        d[k][0] = q.x; d[k][V - 1] = q.y;
      } else {
#pragma unroll
        for (int m = 0; m < V; ++m)
          if (i0 + m < nx) d[k][m] = out[k][g * stride_dst + i0 + m];
      }
    }
  }
  if (in_range) {
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      if (V == 2 && full) {
        const double2 q = *reinterpret_cast<const double2*>(in[k] + g * stride_src + i0);
        u[k][0] = q.x; u[k][V - 1] = q.y;
      } else {
#pragma unroll
        for (int m = 0; m < V; ++m) {
          const long long i = i0 + m;
          const long long j = bc == 0 ? (i % nx + nx) % nx : (i < 0 ? 0 : (i >= nx ? nx - 1 : i));
          u[k][m] = in[k][g * stride_src + j];
        }
      }
    }
  }
#pragma unroll
  for (int m = 0; m < V; ++m) {
    double f[4] = {0.0, 0.0, 0.0, 0.0};
    if (in_range) transport_flux(closure, u[0][m], u[1][m], u[2][m], u[3][m], c, chat, f);
#pragma unroll
    for (int k = 0; k < 4; ++k) { s_u[k][V * t + m] = u[k][m]; s_f[k][V * t + m] = f[k]; }
  }
  __syncthreads();
  if (writer) {
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      double r[V];
#pragma unroll
      for (int m = 0; m < V; ++m) {
        const int a = V * t + m;
        const double fl = 0.5 * (s_f[k][a - 1] + s_f[k][a]) - 0.5 * chat * (s_u[k][a] - s_u[k][a - 1]);
        const double fr = 0.5 * (s_f[k][a] + s_f[k][a + 1]) - 0.5 * chat * (s_u[k][a + 1] - s_u[k][a]);
        r[m] = d[k][m] + -wdt_over_dx * (fr - fl);
      }
      if (V == 2 && full) {
        *reinterpret_cast<double2*>(out[k] + g * stride_dst + i0) = make_double2(r[0], r[V - 1]);
      } else {
#pragma unroll
        for (int m = 0; m < V; ++m)
          if (i0 + m < nx) out[k][g * stride_dst + i0 + m] = r[m];
      }
    }
  }
}

// a = (a + b)/2, element-wise (stage 2 of Eq. 36: (U^n + U^(n+1/2))/2).
__global__ void average_kernel(double* __restrict__ a, const double* __restrict__ b, long long n) {
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
    a[i] = 0.5 * (a[i] + b[i]);
}

}  // namespace mgrhd
