// mgrhd_general.cuh -- the general kernel of the implicit source update: one WARP
// per cell, lane j owns the GPL consecutive groups g = j*GPL .. j*GPL + GPL-1, everything in registers.
//
// It exists for the model options whose group evaluation needs the values of NEIGHBOURING groups and
// therefore does not fit the tuned kernel's lanes-per-cell state machine (mgrhd_kernels.cuh):
//   * the PPL free-slope spectrum fit of Appendix A (Eq. A1-A2): alpha_B,g and
//     alpha_E,g from the group integrals of the two neighbours, refitted at every Newton evaluation,
//     chi_B != chi_E from Eq. 30;
//   * opacity_kind 2: opacities tabulated at the group EDGES in ln T, alpha_g from the two edge values
//     of the group (Eq. 20) at every trial temperature.
// With lane = group a neighbour is one shuffle away and the sums of Eq. 48-52 are full-warp butterflies.
// It also runs every other option (opacity_kind 0/1, S_g), which the tests use to cross-check the two
// kernels.  The iteration (iterates, stopping tests, guards, readings S8-S10, S19-S21 of DESIGN.md) is the
// same as the tuned kernel's; the Planck edge functions (row form) and the closure are the same device functions.
//
// Cost: every lane of a warp evaluates a different edge (hence the per-interval rows of planck_edge_t: a
// three-branch evaluation would run every branch in every evaluation), and a cell's 4 Nq + 5 loads touch
// 4 Nq + 5 different sectors (cell index is the fastest in the state): a feature path, measured separately
// (DESIGN.md section 12), not the benchmark path.
//
// Product code; shares nothing with oracle/.
#pragma once
#include "mgrhd_kernels.cuh"

namespace mgrhd {

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
  return v;
}

// [ (r^q - 1)/q ] of Eq. 30, ln r at q ln r = 0.  Out of line: four uses per group.
__device__ __noinline__ double eq30_bracket(double q, double lnr) {
  const double z = q * lnr;
  return z == 0.0 ? lnr : expm1(z) / q;
}

// One out-of-line copy of the row evaluation (two call sites per evaluation).
__device__ __noinline__ EdgeOut planck_edge_t_call(double x, const double* rows) {
  EdgeOut o;
  bool sm;
  planck_edge_t(x, rows, o.yz, o.xi, sm, o.flops);
  o.small = sm;
  return o;
}

// minmod of Eq. A2.
__device__ __forceinline__ double minmod(double a, double b) {
  if (a * b <= 0.0) return 0.0;
  return fabs(a) < fabs(b) ? a : b;
}

// Eq. A1-A2 for the lane's groups: Q[k] group integrals (all lanes call; converged warp).
//   alpha_Q,g = minmod(s_{g-1/2}, s_{g+1/2}), s_{g+1/2} = ln(Qbar_{g+1}/Qbar_g)/ln(nubar_{g+1}/nubar_g);
//   edge groups, and groups next to a non-positive Q or an open group, get -1 (reading S21).
template <int GPL>
__device__ __forceinline__ void free_slopes(const GenParams& G, int Nq, int lane, const double (&Q)[GPL],
                                            double (&aQ)[GPL]) {
  const unsigned FULL = 0xffffffffu;
  double qb[GPL], s_up[GPL];
  bool ok_up[GPL];
#pragma unroll
  for (int k = 0; k < GPL; ++k) {
    const int g = lane * GPL + k;
    qb[k] = g < Nq ? Q[k] / G.width[g < Nq ? g : 0] : 0.0;
  }
  const double qb_right = __shfl_down_sync(FULL, qb[0], 1);           // first group of the lane to the right
#pragma unroll
  for (int k = 0; k < GPL; ++k) {
    const int g = lane * GPL + k;
    const double qn = k + 1 < GPL ? qb[k + 1 < GPL ? k + 1 : 0] : qb_right;
    const double il = g + 1 < Nq ? G.inv_lnnb[g] : 0.0;
    ok_up[k] = g + 1 < Nq && qb[k] > 0.0 && qn > 0.0 && il != 0.0 && !(lane == 31 && k == GPL - 1);
    s_up[k] = ok_up[k] ? log(qn / qb[k]) * il : 0.0;
  }
  const double s_left = __shfl_up_sync(FULL, s_up[GPL - 1], 1);       // s_{g-1/2} of the lane's first group
  const int ok_left = __shfl_up_sync(FULL, (int)ok_up[GPL - 1], 1);
#pragma unroll
  for (int k = 0; k < GPL; ++k) {
    const int g = lane * GPL + k;
    const double sd = k > 0 ? s_up[k > 0 ? k - 1 : 0] : s_left;
    const bool okd = k > 0 ? ok_up[k > 0 ? k - 1 : 0] : (lane > 0 && ok_left != 0);
    const bool interior = g >= 1 && g + 1 < Nq;
    aQ[k] = interior && okd && ok_up[k] ? minmod(sd, s_up[k]) : -1.0;
  }
}

// The closure's pressure tensor in the form P^{ji} = Pa delta_ji + Pb t_j t_i (reading S7; t = F/(cE) scaled as in
// closure_vP, Pb = 0 on the isotropic lanes), for the implicit-in-v outer stage.
__device__ __forceinline__ void closure_P(int closure, double E, double F0, double F1, double F2, double c,
                                          double& Pa, double& Pb, double& t0, double& t1, double& t2) {
  const double cE0 = c * E;
  const double sc = cE0 < 1e-200 ? 0x1p+400 : (cE0 > 1e200 ? 0x1p-400 : 1.0);
  const double cE = cE0 * sc;
  const bool Fzero = fma(F0, F0, fma(F1, F1, F2 * F2)) == 0.0;
  const double r1 = 1.0 / (cE > 0.0 ? cE : 1.0);
  t0 = F0 * sc * r1; t1 = F1 * sc * r1; t2 = F2 * sc * r1;
  const double f2u = fma(t0, t0, fma(t1, t1, t2 * t2));
  const bool iso = closure == 1 || !(E > 0.0) || Fzero || !(f2u > 1e-290) || !(f2u < 1e290);
  const double f2 = f2u > 1.0 ? 1.0 : f2u;
  const double sq = sqrt(fma(-3.0, f2, 4.0));
  Pa = iso ? E * (1.0 / 3.0) : E * ((sq - 1.0) * (1.0 / 3.0));
  Pb = iso ? 0.0 : E * ((2.0 - sq) / f2u);
  if (iso) { t0 = 0.0; t1 = 0.0; t2 = 0.0; }
}

enum GenStat : int { GS_EVALS = 0, GS_TRIPS, GS_GUARD, GS_DEN, GS_COUNT };

// GPL: groups per lane (1: Nq <= 32, 2: Nq <= 64).  256 threads = 8 warps = 8 cells in flight per CTA.
// COUNT: the instrumented instantiation also sums the algorithmic flops of DESIGN.md section 8 (with the general
// kernel's rows for the free-slope fit, the tabulated opacities and the implicit-in-v outer stage) into kStatFlops.
template <int GPL, bool COUNT>
__global__ void __launch_bounds__(256)
source_update_general_kernel(const __grid_constant__ Params P, const __grid_constant__ GenParams G,
                             const __grid_constant__ StatePtrs S, unsigned long long* __restrict__ stats) {
  __shared__ unsigned int s_hist[2 * MGRHD_HIST];
  __shared__ unsigned int s_cnt[GS_COUNT];
  __shared__ __align__(16) double s_rows[kRows * kRowStride];     // per-interval rows of the edge functions
  for (int t = threadIdx.x; t < kRows * kRowStride; t += blockDim.x) s_rows[t] = mgrhd_g_rows[t];
  for (int t = threadIdx.x; t < 2 * MGRHD_HIST; t += blockDim.x) s_hist[t] = 0u;
  if (threadIdx.x < GS_COUNT) s_cnt[threadIdx.x] = 0u;
  __syncthreads();

  const unsigned FULL = 0xffffffffu;
  const int lane = threadIdx.x & 31;
  const int Nq = P.Nq;
  const long long n = P.ncells, stride = P.stride;
  const double dt = P.dt, c = P.c, chat = P.c_hat;
  const double c_over_chat = c / chat, cdt = chat * dt, icc = 1.0 / (c * chat), inv_c = 1.0 / c, inv_cdt = 1.0 / cdt;
  const double NaN = __longlong_as_double(0x7ff8000000000000ll);
  const long long nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
  const long long warp0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;

  // per-group constants of the lane's groups
  int gi[GPL];
  bool vg[GPL];
  double nu_hi[GPL], lnr[GPL], k_lo[GPL], k_hi[GPL], al_tab[GPL];
#pragma unroll
  for (int k = 0; k < GPL; ++k) {
    const int g = lane * GPL + k;
    vg[k] = g < Nq;
    gi[k] = vg[k] ? g : 0;
    nu_hi[k] = P.nu[gi[k] + 1];
    lnr[k] = G.lnr[gi[k]];
    k_lo[k] = P.k_lo[gi[k]];
    k_hi[k] = P.k_hi[gi[k]];
    al_tab[k] = P.alpha[gi[k]];
  }

  // algorithmic flops of one group at one trial T beyond the edge functions, and of one cell
  unsigned long long flops = 0;
  const bool varmeans = G.opacity_kind == 2 || G.spectrum == 1;   // chi_B, chi_E change with the iterate
  const int fl_group = kFlopGroupEval + (G.opacity_kind == 2 ? kFlopTabEdge + kFlopTabAlpha : 0) +
                       (varmeans ? kFlopMeansVar : 0) + (G.spectrum == 1 ? 2 * kFlopSlopeFit : 0);
  const int fl_eq30 = G.spectrum == 1 ? 2 * kFlopEq30Free : (G.opacity_kind == 2 ? kFlopEq30Fixed : 0);
  const int fl_cell = kFlopCellEval + (G.opacity_kind == 1 ? kFlopPowT : 0) +
                      (G.opacity_kind == 2 ? kFlopTabCell + kFlopTabEdge : 0);

  for (long long cell = warp0; cell < n; cell += nwarps) {
    // ---- a0: load (the post-explicit state U^(t)) --------------------------------------
    const double rho = S.rho[cell];
    const double ks = S.kappa_scale ? S.kappa_scale[cell] : 1.0;
    const double momt0 = S.mom[0][cell], momt1 = S.mom[1][cell], momt2 = S.mom[2][cell];
    const double Egas_t = S.Egas[cell];
    const double chis = rho * ks, inv_rho = 1.0 / rho;
    const double Cv = rho * P.cv_over_rho, inv_Cv = 1.0 / Cv;
    double Et[GPL], Sg[GPL], R[GPL], Ft0[GPL], Ft1[GPL], Ft2[GPL], Fk0[GPL], Fk1[GPL], Fk2[GPL];
    double Fn0[GPL], Fn1[GPL], Fn2[GPL], Enew[GPL];
    double sumEtS = 0.0;
#pragma unroll
    for (int k = 0; k < GPL; ++k) {
      const long long o = (long long)gi[k] * stride + cell;
      Et[k] = vg[k] ? S.Erad[o] : 0.0;
      Sg[k] = vg[k] && S.Srad ? S.Srad[o] : 0.0;
      Ft0[k] = vg[k] ? S.Frad[0][o] : 0.0; Ft1[k] = vg[k] ? S.Frad[1][o] : 0.0; Ft2[k] = vg[k] ? S.Frad[2][o] : 0.0;
      Fk0[k] = Ft0[k]; Fk1[k] = Ft1[k]; Fk2[k] = Ft2[k];
      Fn0[k] = Ft0[k]; Fn1[k] = Ft1[k]; Fn2[k] = Ft2[k];
      R[k] = 0.0;
      Enew[k] = Et[k];
      sumEtS += Et[k] + Sg[k];
    }
    const double Etot = Egas_t + (chat / c) * warp_sum(sumEtS);        // Eq. 50 as printed
    if (COUNT && lane == 0) flops += kFlopCell + kFlopCellGroup * Nq;
    double momk0 = momt0, momk1 = momt1, momk2 = momt2, momn0 = momt0, momn1 = momt1, momn2 = momt2;
    double Egs = Egas_t, Egas_new = Egas_t;
    int evals = 0, trips = 0;
    // group quantities of the last evaluation (used by Eq. 51 and the outer test)
    double alpha[GPL], chiE[GPL], chiF[GPL], AG[GPL], W[GPL];

    for (int kk = 0; kk < P.outer_maxit; ++kk) {
      // ---- O1: lagged velocity and fluxes -------------------------------------------
      const double v0 = momk0 * inv_rho, v1 = momk1 * inv_rho, v2 = momk2 * inv_rho;
      const double Ekin = (momk0 * momk0 + momk1 * momk1 + momk2 * momk2) * (0.5 * inv_rho);
      double vF[GPL];
#pragma unroll
      for (int k = 0; k < GPL; ++k) vF[k] = fma(v0, Fk0[k], fma(v1, Fk1[k], v2 * Fk2[k]));
      if (!((Egs - Ekin) * inv_Cv > 0.0)) {                              // invalid state: stop here (S9)
        if (lane == 0) atomicAdd(&stats[kStatTNonPos], 1ull);
        break;
      }
      // ---- inner Newton-Raphson iteration on x = (E_gas, R_1..R_Nq) (Eq. 41-50) ---------------------
      for (int it = 0;; ++it) {
        const double T = (Egs - Ekin) * inv_Cv;
        const double invT = 1.0 / T;
        const double T2 = T * T, aT4 = P.a_rad * T2 * T2;
        const double beta = P.h_over_k * invT;
        // a1: edge functions at the lane's upper edges; the lower edge comes from the left, edge 0 from an
        // evaluation of its own (lane 0).  The 32 lanes hold 32 different x, so the per-interval rows
        // (planck_edge_t: one row per lane, no branch but e^-x) replace three warp-wide branches per evaluation.
        double hy[GPL], hx[GPL], ly[GPL], lx[GPL];
        bool hs[GPL], ls[GPL];
#pragma unroll 1
        for (int k = 0; k < GPL; ++k) {
          const EdgeOut o = planck_edge_t_call(vg[k] ? nu_hi[k] * beta : NaN, s_rows);
          hy[k] = o.yz; hx[k] = o.xi; hs[k] = o.small != 0;
          if (COUNT && vg[k]) flops += o.flops;
        }
        double e0y, e0x;
        bool e0s;
        {
          const EdgeOut o = planck_edge_t_call(lane == 0 ? P.nu[0] * beta : NaN, s_rows);
          e0y = o.yz; e0x = o.xi; e0s = o.small != 0;
          if (COUNT && lane == 0) flops += o.flops;
        }
        {
          const double uy = __shfl_up_sync(FULL, hy[GPL - 1], 1), ux = __shfl_up_sync(FULL, hx[GPL - 1], 1);
          const int us = __shfl_up_sync(FULL, (int)hs[GPL - 1], 1);
#pragma unroll
          for (int k = 0; k < GPL; ++k) {
            ly[k] = k > 0 ? hy[k > 0 ? k - 1 : 0] : (lane == 0 ? e0y : uy);
            lx[k] = k > 0 ? hx[k > 0 ? k - 1 : 0] : (lane == 0 ? e0x : ux);
            ls[k] = k > 0 ? hs[k > 0 ? k - 1 : 0] : (lane == 0 ? e0s : us != 0);
          }
        }
        // a2: group Planck integrals per unit a_R T^4 (Eq. 11): no cancellation in the Wien tail
        double dY[GPL], dX[GPL], Bt[GPL];
#pragma unroll
        for (int k = 0; k < GPL; ++k) {
          dY[k] = hs[k] ? hy[k] - ly[k] : (ls[k] ? (1.0 - ly[k]) - hy[k] : ly[k] - hy[k]);
          dX[k] = hx[k] - lx[k];
          Bt[k] = vg[k] ? aT4 * dY[k] : 0.0;
        }
        // a3: opacities at the group edges at this trial temperature (Eq. 19, 20)
        double chi_lo[GPL], chi_hi[GPL];
        if (G.opacity_kind == 2) {
          const double lnT = log(T);
          double u = (lnT - G.lnT0) * G.inv_dlnT;
          if (!(u > 0.0)) u = 0.0;
          if (u > (double)(G.NT - 1)) u = (double)(G.NT - 1);
          int j = (int)u;
          if (j > G.NT - 2) j = G.NT - 2;
          if (j < 0) j = 0;
          const double w = G.NT > 1 ? u - (double)j : 0.0;
          auto edge_chi = [&](int e) {
            const double* row = G.lnk_edge + (long long)e * G.NT;
            const double lnk = G.NT > 1 ? (1.0 - w) * row[j] + w * row[j + 1] : row[0];
            return chis * exp(lnk);
          };
#pragma unroll
          for (int k = 0; k < GPL; ++k) chi_hi[k] = edge_chi(gi[k] + 1);
          const double c0 = edge_chi(0);
          const double cu = __shfl_up_sync(FULL, chi_hi[GPL - 1], 1);
#pragma unroll
          for (int k = 0; k < GPL; ++k) {
            chi_lo[k] = k > 0 ? chi_hi[k > 0 ? k - 1 : 0] : (lane == 0 ? c0 : cu);
            alpha[k] = log(chi_hi[k] / chi_lo[k]) / lnr[k];                        // Eq. 20
          }
        } else {
          const double f = G.opacity_kind == 1 ? exp(P.p_T * log(T * P.inv_T_ref)) : 1.0;
#pragma unroll
          for (int k = 0; k < GPL; ++k) {
            alpha[k] = al_tab[k];
            chi_lo[k] = chis * k_lo[k] * f;
            chi_hi[k] = chis * k_hi[k] * f;                                        // Eq. 19 at nu_g+
          }
        }
        // spectrum slopes alpha_B,g, alpha_E,g (fixed: -1; free: Appendix A, refitted from B_g at
        // this T and from the current iterate E_g^(t) + R_g + S_g, reading S20) and the means of Eq. 30
        double aB[GPL], aE[GPL], chiB[GPL];
#pragma unroll
        for (int k = 0; k < GPL; ++k) { aB[k] = -1.0; aE[k] = -1.0; }
        if (G.spectrum == 1) {
          double Ecur[GPL];
#pragma unroll
          for (int k = 0; k < GPL; ++k) Ecur[k] = Et[k] + R[k] + Sg[k];
          free_slopes<GPL>(G, Nq, lane, Bt, aB);
          free_slopes<GPL>(G, Nq, lane, Ecur, aE);
        }
        double sumR = 0.0, sumAbsFR = 0.0, SFRq = 0.0, SJq = 0.0, FR[GPL], qg[GPL], jg0[GPL];
        unsigned n_guard = 0, n_den = 0;
#pragma unroll
        for (int k = 0; k < GPL; ++k) {
          if (alpha[k] == 0.0) {
            chiB[k] = chi_lo[k];                                                   // PC, Eq. 17
            chiE[k] = chi_lo[k];
          } else {
            // Eq. 30; the second bracket is ln r for alpha_Q = -1, and with the fixed slope chi_E = chi_B
            const double bB = aB[k] + 1.0;
            chiB[k] = chi_lo[k] * eq30_bracket(alpha[k] + bB, lnr[k]) / (bB == 0.0 ? lnr[k] : eq30_bracket(bB, lnr[k]));
            chiE[k] = chiB[k];
            if (G.spectrum == 1) {
              const double bE = aE[k] + 1.0;
              chiE[k] = chi_lo[k] * eq30_bracket(alpha[k] + bE, lnr[k]) / (bE == 0.0 ? lnr[k] : eq30_bracket(bE, lnr[k]));
            }
          }
          // a2: Doppler boundary term Delta_g(nu chi_0 B_nu) per unit a_R T^4 (Eq. 22)
          const double P3 = fma(chi_hi[k], hx[k], -chi_lo[k] * lx[k]);
          const double fbd = fma(4.0, dY[k], -dX[k]);                              // 3 x denominator of Eq. 27
          // a3: flux-mean opacity, Eq. 27, with the guards of reading S8
          const bool guard = !(fbd >= 3e-280) || isinf(aT4 * fbd);
          double cf = (fma(3.0 * chiB[k] + (1.0 + alpha[k]) * chiE[k], dY[k], -P3)) / (guard ? 1.0 : fbd);
          if (guard) cf = chi_lo[k];
          const bool denbad = !(fma(cdt, cf, 1.0) > 0.0);
          if (denbad) cf = chiE[k];
          if (vg[k] && evals == 0) { n_guard += guard ? 1u : 0u; n_den += denbad ? 1u : 0u; }
          chiF[k] = cf;
          if (COUNT && vg[k]) flops += fl_group + (alpha[k] != 0.0 ? fl_eq30 : 0);
          // a4: work term, Eq. 42 solved for E_g, residuals of Eq. 41
          W[k] = (1.0 + alpha[k]) * cf * vF[k] * inv_c;
          const double inv_chiE = 1.0 / chiE[k];
          const double ratio = chiB[k] * inv_chiE;
          const double itau = inv_cdt * inv_chiE;                                   // 1/(c_hat dt chi_E)
          const double Eg = fma(ratio, Bt[k], W[k] * (inv_c * inv_chiE)) - R[k] * itau;
          FR[k] = vg[k] ? Eg - Et[k] - (R[k] + Sg[k]) : 0.0;
          // a5: Jacobian, Eq. 44-47 (d(chi_B/chi_E)/dT = 0), q = -1/J_gg
          qg[k] = 1.0 / (itau + 1.0);
          jg0[k] = ratio * (aT4 * fbd * invT) * inv_Cv;                            // (4 Bt - Db)/T / C_v
          AG[k] = aT4 * fma(chiB[k], dY[k], P3 * (-1.0 / 3.0));                    // chi_B Bt - D/3 (Eq. 51 source)
          if (vg[k]) {
            sumR += R[k];
            sumAbsFR += fabs(FR[k]);
            SFRq += FR[k] * qg[k];
            SJq += jg0[k] * qg[k];
          }
        }
        sumR = warp_sum(sumR); sumAbsFR = warp_sum(sumAbsFR); SFRq = warp_sum(SFRq); SJq = warp_sum(SJq);
        if (evals == 0) {
          const unsigned ng = __reduce_add_sync(FULL, n_guard), nd = __reduce_add_sync(FULL, n_den);
          if (lane == 0 && ng) atomicAdd(&s_cnt[GS_GUARD], ng);
          if (lane == 0 && nd) atomicAdd(&s_cnt[GS_DEN], nd);
        }
        const double FG = Egs - Egas_t + c_over_chat * sumR;
        evals++;
        if (COUNT && lane == 0) flops += fl_cell;
        // Eq. 49
        if (fabs(FG) / Etot < P.newton_tol && c_over_chat * sumAbsFR / Etot < P.newton_tol) break;
        if (it >= P.newton_maxit) {
          if (lane == 0) atomicAdd(&stats[kStatNewtonUnconv], 1ull);
          break;
        }
        // Newton step: eliminate the gas row of the arrowhead Jacobian (Eq. 48)
        const double dx0 = (-FG - c_over_chat * SFRq) / fma(c_over_chat, SJq, 1.0);
        double lam = 1.0;
#pragma unroll 1
        for (int h = 0; h < 10 && !((Egs + lam * dx0 - Ekin) * inv_Cv > 0.0); ++h) {   // S9
          lam *= 0.5;
          if (lane == 0) atomicAdd(&stats[kStatTNonPos], 1ull);
        }
        Egs += lam * dx0;
#pragma unroll
        for (int k = 0; k < GPL; ++k) R[k] += lam * (FR[k] + jg0[k] * dx0) * qg[k];
        if (COUNT && lane == 0) flops += kFlopStepCell + kFlopStepGroup * Nq;
      }

      // ---- a6: energy commit ---------------------------------------------------------
      double sR = 0.0, sAbsR = 0.0;
#pragma unroll
      for (int k = 0; k < GPL; ++k) {
        Enew[k] = Et[k] + R[k] + Sg[k];
        if (vg[k]) { sR += R[k]; sAbsR += fabs(R[k]); }
      }
      sR = warp_sum(sR); sAbsR = warp_sum(sAbsR);
      Egas_new = Egas_t - c_over_chat * sR;
      // ---- a7: closure + flux update with the lagged velocity (Eq. 51); a8: gas momentum (Eq. 52) ----
      double dF0 = 0.0, dF1 = 0.0, dF2 = 0.0;
      bool rel_ok = true;
      if (G.outer_mode == 1) {
        // "variant L": v in Eq. 51 is the NEW velocity: F_g^new = a_g + B_g v^new with a_g = F_g^t/dn_g,
        // B_g = (c_hat dt/dn_g)[(chi_B Bt - D/3) I + (1 + alpha) chi_E P_g], and Eq. 52 becomes the 3x3 system
        //   [rho I + (c c_hat)^-1 sum_g B_g] v^new = (rho v)^t - (c c_hat)^-1 sum_g (a_g - F_g^t)
        double ca[GPL], cb[GPL], tt0[GPL], tt1[GPL], tt2[GPL], idn[GPL];
        double m00 = 0, m01 = 0, m02 = 0, m11 = 0, m12 = 0, m22 = 0, r0 = 0, r1 = 0, r2 = 0;
#pragma unroll
        for (int k = 0; k < GPL; ++k) {
          double Pa, Pb;
          closure_P(P.closure, Enew[k], Fk0[k], Fk1[k], Fk2[k], c, Pa, Pb, tt0[k], tt1[k], tt2[k]);
          const double w = (1.0 + alpha[k]) * chiE[k];
          idn[k] = 1.0 / fma(cdt, chiF[k], 1.0);
          ca[k] = cdt * idn[k] * fma(w, Pa, AG[k]);       // isotropic part of B_g
          cb[k] = cdt * idn[k] * (w * Pb);                // coefficient of t t^T
          if (vg[k]) {
            m00 += fma(cb[k], tt0[k] * tt0[k], ca[k]); m11 += fma(cb[k], tt1[k] * tt1[k], ca[k]); m22 += fma(cb[k], tt2[k] * tt2[k], ca[k]);
            m01 += cb[k] * tt0[k] * tt1[k]; m02 += cb[k] * tt0[k] * tt2[k]; m12 += cb[k] * tt1[k] * tt2[k];
            r0 += Ft0[k] * idn[k] - Ft0[k]; r1 += Ft1[k] * idn[k] - Ft1[k]; r2 += Ft2[k] * idn[k] - Ft2[k];
          }
        }
        m00 = fma(icc, warp_sum(m00), rho); m11 = fma(icc, warp_sum(m11), rho); m22 = fma(icc, warp_sum(m22), rho);
        m01 = icc * warp_sum(m01); m02 = icc * warp_sum(m02); m12 = icc * warp_sum(m12);
        r0 = momt0 - icc * warp_sum(r0); r1 = momt1 - icc * warp_sum(r1); r2 = momt2 - icc * warp_sum(r2);
        // symmetric 3x3 solve by cofactors
        const double c00 = m11 * m22 - m12 * m12, c01 = m02 * m12 - m01 * m22, c02 = m01 * m12 - m02 * m11;
        const double c11 = m00 * m22 - m02 * m02, c12 = m01 * m02 - m00 * m12, c22 = m00 * m11 - m01 * m01;
        const double idet = 1.0 / (m00 * c00 + m01 * c01 + m02 * c02);
        const double w0 = (c00 * r0 + c01 * r1 + c02 * r2) * idet, w1 = (c01 * r0 + c11 * r1 + c12 * r2) * idet,
                     w2 = (c02 * r0 + c12 * r1 + c22 * r2) * idet;
#pragma unroll
        for (int k = 0; k < GPL; ++k) {
          const double tv = cb[k] * fma(tt0[k], w0, fma(tt1[k], w1, tt2[k] * w2));
          Fn0[k] = fma(Ft0[k], idn[k], fma(ca[k], w0, tv * tt0[k]));
          Fn1[k] = fma(Ft1[k], idn[k], fma(ca[k], w1, tv * tt1[k]));
          Fn2[k] = fma(Ft2[k], idn[k], fma(ca[k], w2, tv * tt2[k]));
        }
      }
#pragma unroll
      for (int k = 0; k < GPL; ++k) {
        double p0, p1, p2;
        if (G.outer_mode != 1) {
        closure_vP(P.closure, Enew[k], Fk0[k], Fk1[k], Fk2[k], v0, v1, v2, c, p0, p1, p2);
        const double w = (1.0 + alpha[k]) * chiE[k];
        const double dn = fma(cdt, chiF[k], 1.0);
        const double inv_dn = 1.0 / dn;
        Fn0[k] = fma(cdt, fma(v0, AG[k], w * p0), Ft0[k]) * inv_dn;
        Fn1[k] = fma(cdt, fma(v1, AG[k], w * p1), Ft1[k]) * inv_dn;
        Fn2[k] = fma(cdt, fma(v2, AG[k], w * p2), Ft2[k]) * inv_dn;
        }
        if (vg[k]) {
          dF0 += Fn0[k] - Ft0[k]; dF1 += Fn1[k] - Ft1[k]; dF2 += Fn2[k] - Ft2[k];
          if (P.outer_stop == 1 &&
              !(norm3(Fn0[k] - Fk0[k], Fn1[k] - Fk1[k], Fn2[k] - Fk2[k]) <= P.outer_rel_tol * norm3(Fn0[k], Fn1[k], Fn2[k])))
            rel_ok = false;
        }
      }
      dF0 = warp_sum(dF0); dF1 = warp_sum(dF1); dF2 = warp_sum(dF2);
      momn0 = momt0 - dF0 * icc; momn1 = momt1 - dF1 * icc; momn2 = momt2 - dF2 * icc;
      trips++;
      if (COUNT && lane == 0)
        flops += G.outer_mode == 1 ? kFlopOuterCellL + kFlopOuterGroupL * Nq : kFlopOuterCell + kFlopOuterGroup * Nq;
      // ---- a9: outer test (reading S10) ------------------------------------------------
      const double vn0 = momn0 * inv_rho, vn1 = momn1 * inv_rho, vn2 = momn2 * inv_rho;
      double dW = 0.0;
#pragma unroll
      for (int k = 0; k < GPL; ++k) {
        const double vFn = fma(vn0, Fn0[k], fma(vn1, Fn1[k], vn2 * Fn2[k]));
        const double Wn = (1.0 + alpha[k]) * chiF[k] * vFn * inv_c;
        if (vg[k]) dW += fabs(Wn - W[k]);
      }
      dW = warp_sum(dW);
      rel_ok = __all_sync(FULL, rel_ok);
      if (P.outer_stop == 1 &&
          !(norm3(momn0 - momk0, momn1 - momk1, momn2 - momk2) <= P.outer_rel_tol * norm3(momn0, momn1, momn2)))
        rel_ok = false;
      const double delta = dW * (chat / c) * dt;
      if (delta <= P.outer_tol * fmax(sAbsR, Etot) && rel_ok) break;
      if (kk == P.outer_maxit - 1) {
        if (lane == 0) atomicAdd(&stats[kStatOuterUnconv], 1ull);
        break;
      }
      momk0 = momn0; momk1 = momn1; momk2 = momn2;
#pragma unroll
      for (int k = 0; k < GPL; ++k) { Fk0[k] = Fn0[k]; Fk1[k] = Fn1[k]; Fk2[k] = Fn2[k]; }
    }

    // ---- a10: store in place ------------------------------------------------------------------------
    if (trips > 0) {
      if (lane == 0) {
        S.mom[0][cell] = momn0; S.mom[1][cell] = momn1; S.mom[2][cell] = momn2;
        S.Egas[cell] = Egas_new;     // total gas energy; E_int = Egas - |mom|^2/(2 rho)
      }
#pragma unroll
      for (int k = 0; k < GPL; ++k)
        if (vg[k]) {
          const long long o = (long long)gi[k] * stride + cell;
          S.Erad[o] = Enew[k];
          S.Frad[0][o] = Fn0[k]; S.Frad[1][o] = Fn1[k]; S.Frad[2][o] = Fn2[k];
        }
    }
    if (lane == 0) {
      atomicAdd(&s_cnt[GS_EVALS], (unsigned)evals);
      atomicAdd(&s_cnt[GS_TRIPS], (unsigned)trips);
      atomicAdd(&s_hist[evals < MGRHD_HIST ? evals : MGRHD_HIST - 1], 1u);
      atomicAdd(&s_hist[MGRHD_HIST + (trips < MGRHD_HIST ? trips : MGRHD_HIST - 1)], 1u);
    }
  }

  if (COUNT) {
    for (int off = 16; off > 0; off >>= 1) flops += __shfl_xor_sync(FULL, flops, off);
    if (lane == 0) atomicAdd(&stats[kStatFlops], flops);
  }
  __syncthreads();
  if (threadIdx.x < GS_COUNT && s_cnt[threadIdx.x]) {
    const int t = threadIdx.x;
    const int slot = t == GS_EVALS ? kStatNewtonEvals : (t == GS_TRIPS ? kStatOuterTrips : (t == GS_GUARD ? kStatChiFGuard : kStatDenNonPos));
    atomicAdd(&stats[slot], (unsigned long long)s_cnt[t]);
  }
  for (int t = threadIdx.x; t < 2 * MGRHD_HIST; t += blockDim.x)
    if (s_hist[t]) {
      atomicAdd(&stats[kStatNewtonHist + t], (unsigned long long)s_hist[t]);
      if (t < MGRHD_HIST) atomicAdd(&stats[kStatCells], (unsigned long long)s_hist[t]);
    }
}

}  // namespace mgrhd
