// mgrhd_kernels.cuh -- the per-cell implicit source update (Eq. 37-52)
// as one persistent CUDA kernel: one THREAD owns one cell from load to store.
//
// Mapping:
//  * thread-per-cell, because the dominant cost is the Planck edge functions at the Nq+1
//    group edges, re-evaluated at every trial temperature: with one cell per thread the EDGE
//    index is warp-uniform, so 32 lanes evaluate the same edge at 32 temperatures and almost
//    always take the same branch of planck_edge(); with lanes mapped to groups every warp
//    would execute every branch.
//  * per-(cell,group) iteration state lives in SHARED memory, laid out [slot][group][thread]
//    (conflict-free 8-byte lanes); the lagged fluxes F_g,k live in a small per-thread global
//    scratch that stays L2-resident.  Nothing is spilled to local memory.
//  * the Newton loop inside the outer loop is FLATTENED into one loop whose body is
//    "evaluate all groups at the trial T", followed by a cheap Newton step or by the
//    flux/momentum update; a lane whose cell has converged stores it and takes the next cell
//    of its warp's contiguous chunk at once (no atomics), so unequal iteration counts do not
//    leave lanes idle: every live lane does one full-width evaluation per loop trip.
//
// Product code; shares nothing with oracle/.
#pragma once
#include "mgrhd_planck.cuh"

namespace mgrhd {

// ---- fast, IEEE-faithful-to-1-ulp reciprocal / sqrt for NORMAL positive arguments -----------
// rcp.approx.ftz.f64 gives ~20 bits; two Newton steps give full double precision.  Callers
// guarantee 1e-290 < x < 1e290 (otherwise they take the IEEE path).
__device__ __forceinline__ double fast_rcp(double x) {   // declared in mgrhd_planck.cuh
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  double e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  return r;
}

__device__ __forceinline__ double norm3(double a, double b, double c) {
  return sqrt(fma(a, a, fma(b, b, c * c)));
}

// v^j P^{ji} for one group (closure reading S7 of DESIGN.md): Levermore/M1
// or Eddington P = E/3 I.
__device__ __forceinline__ void closure_vP(int closure, double E, double F0, double F1, double F2,
                                           double v0, double v1, double v2, double c,
                                           double& p0, double& p1, double& p2) {
  const double Fn = norm3(F0, F1, F2);
  if (closure == 1 || !(E > 0.0) || Fn == 0.0) {
    const double t = E * (1.0 / 3.0);
    p0 = t * v0; p1 = t * v1; p2 = t * v2;
    return;
  }
  const double cE = c * E;
  double f, inv_Fn;
  if (cE > 1e-290 && cE < 1e290 && Fn > 1e-290 && Fn < 1e290) {
    f = Fn * fast_rcp(cE);
    inv_Fn = fast_rcp(Fn);
  } else {               // denormal / huge group energies: IEEE division
    f = Fn / cE;
    inv_Fn = 1.0 / Fn;
  }
  if (f > 1.0) f = 1.0;
  const double f2 = f * f;
  const double chi = fma(4.0, f2, 3.0) * fast_rcp(fma(2.0, sqrt(fma(-3.0, f2, 4.0)), 5.0));
  const double n0 = F0 * inv_Fn, n1 = F1 * inv_Fn, n2 = F2 * inv_Fn;
  const double ndv = fma(n0, v0, fma(n1, v1, n2 * v2));
  const double a = 0.5 * (1.0 - chi), b = 0.5 * fma(3.0, chi, -1.0) * ndv;
  p0 = E * fma(a, v0, b * n0);
  p1 = E * fma(a, v1, b * n1);
  p2 = E * fma(a, v2, b * n2);
}

// Lane phases of the flattened iteration.
enum Phase : int { PH_LOAD = 0, PH_EVAL = 1, PH_FLUX = 2, PH_STORE = 3, PH_DONE = 4 };

// Shared-memory slots (per thread, per group).
enum Slot : int { SL_R = 0, SL_DA, SL_DB, SL_VF, SL_AG, SL_CHIF, SL_COUNT };


// NQ: compile-time group capacity (runtime Nq <= NQ); THREADS: CTA size; NSMEM: how many of the
// SL_COUNT per-group slots live in shared memory (the rest go to the global scratch).
// Dynamic shared memory: NSMEM * NQ * THREADS doubles.
// scratch: (3 + SL_COUNT - NSMEM) * NQ * (gridDim.x*THREADS) doubles of global memory (the lagged
// fluxes F_g,k and the overflow slots), private to this launch.
template <int NQ, int THREADS, int NSMEM, bool COUNT>
__global__ void __launch_bounds__(THREADS, 1)
source_update_kernel(const __grid_constant__ Params P, const __grid_constant__ StatePtrs S,
                     unsigned long long* __restrict__ stats, double* __restrict__ scratch) {
  extern __shared__ double smem[];
  __shared__ unsigned int s_hist[2 * MGRHD_HIST];
  for (int t = threadIdx.x; t < 2 * MGRHD_HIST; t += THREADS) s_hist[t] = 0u;
  __syncthreads();

  const int tid = threadIdx.x, lane = tid & 31;
  const unsigned FULL = 0xffffffffu;
  const int Nq = P.Nq;
  const long long n = P.ncells, stride = P.stride;
  const double dt = P.dt, c = P.c, chat = P.c_hat;
  const double c_over_chat = c / chat, inv_c = 1.0 / c, cdt = chat * dt, icc = 1.0 / (c * chat);

  // shared-memory slot s, group g of this thread
  auto sm = [&](int s, int g) -> double& {
    if (s < NSMEM) return smem[(s * NQ + g) * THREADS + tid];
    return scratch[(long long)((3 + s - NSMEM) * NQ + g) * ((long long)gridDim.x * THREADS) +
                   ((long long)blockIdx.x * THREADS + tid)];
  };
  // lagged flux component i, group g of this thread (global scratch, coalesced across the warp)
  const long long tthreads = (long long)gridDim.x * THREADS;
  double* const fk_base = scratch + ((long long)blockIdx.x * THREADS + tid);
  auto fk = [&](int i, int g) -> double& { return fk_base[(long long)(i * NQ + g) * tthreads]; };

  // this warp's contiguous chunk of cells [next, end)
  const long long nwarps = tthreads >> 5, wid = ((long long)blockIdx.x * THREADS + tid) >> 5;
  const long long per = (n + nwarps - 1) / nwarps;
  long long next = wid * per;
  long long end = next + per < n ? next + per : n;
  if (next > n) next = n;

  unsigned int cnt_newton_unconv = 0, cnt_outer_unconv = 0, cnt_Tnonpos = 0, cnt_guard = 0,
               cnt_den = 0, cnt_evals = 0, cnt_trips = 0, cnt_cells = 0;
  unsigned long long flops = 0;

  // ---- per-lane cell state -----------------------------------------------------------------
  int phase = PH_LOAD;
  long long cell = -1;
  double rho = 1.0, chis = 1.0, inv_chis = 1.0, Cv = 1.0, inv_Cv = 1.0, Egas_t = 0.0, Etot = 1.0;
  double momt0 = 0, momt1 = 0, momt2 = 0, momk0 = 0, momk1 = 0, momk2 = 0, momn0 = 0, momn1 = 0, momn2 = 0;
  double Egs = 0.0, Egas_new = 0.0, Ekin = 0.0;
  int it = 0, k = 0, evals = 0, trips = 0;

  while (true) {
    // ===== LOAD: lanes that need a cell take the next ones of the warp's chunk (a0) ===========
    const unsigned need = __ballot_sync(FULL, phase == PH_LOAD);
    if (need) {
      if (phase == PH_LOAD) {
        const long long cnew = next + __popc(need & ((1u << lane) - 1u));
        if (cnew < end) {
          cell = cnew;
          rho = S.rho[cell];
          const double ks = S.kappa_scale ? S.kappa_scale[cell] : 1.0;
          chis = rho * ks;                      // chi_{g-} = chis * k_lo[g]
          inv_chis = 1.0 / chis;
          Cv = rho * P.cv_over_rho;
          inv_Cv = 1.0 / Cv;
          momt0 = S.mom[0][cell]; momt1 = S.mom[1][cell]; momt2 = S.mom[2][cell];
          Egas_t = S.Egas[cell];
          const double inv_rho = 1.0 / rho;
          const double v0 = momt0 * inv_rho, v1 = momt1 * inv_rho, v2 = momt2 * inv_rho;
          double sumEt = 0.0;
          for (int g = 0; g < Nq; ++g) {
            const long long o = (long long)g * stride + cell;
            const double F0 = S.Frad[0][o], F1 = S.Frad[1][o], F2 = S.Frad[2][o];
            sumEt += S.Erad[o];
            fk(0, g) = F0; fk(1, g) = F1; fk(2, g) = F2;
            sm(SL_R, g) = 0.0;
            sm(SL_VF, g) = fma(v0, F0, fma(v1, F1, v2 * F2));   // lagged v.F_g of the first trip
          }
          Etot = Egas_t + (chat / c) * sumEt;   // Eq. 50 as printed, S_g = 0
          momk0 = momn0 = momt0; momk1 = momn1 = momt1; momk2 = momn2 = momt2;
          Egs = Egas_new = Egas_t;
          Ekin = (momk0 * momk0 + momk1 * momk1 + momk2 * momk2) / (2.0 * rho);
          it = 0; k = 0; evals = 0; trips = 0;
          if (COUNT) flops += kFlopCell + kFlopCellGroup * Nq;
          if ((Egs - Ekin) * inv_Cv > 0.0) phase = PH_EVAL;
          else { cnt_Tnonpos++; phase = PH_STORE; }     // invalid state: leave the cell as it is
        } else {
          phase = PH_DONE;
          cell = -1;
        }
      }
      next += __popc(need);
    }
    if (__all_sync(FULL, phase == PH_DONE)) break;

    // ===== EVAL: all groups at the trial temperature (a1-a5), then Eq. 49 ========================
    if (phase == PH_EVAL) {
      const double T = (Egs - Ekin) * inv_Cv;
      const double invT = 1.0 / T;
      const double T2 = T * T;
      const double aT4 = P.a_rad * T2 * T2;
      const double beta = P.h_over_k * invT;
      const double itau_c = inv_chis / cdt;          // 1/(c_hat dt chi_E,g) = itau_c * inv_k_mean[g]
      const double dBscale = invT * inv_Cv;          // J_g0 = (4 Bt - Db) / (T C_v), Eq. 46
      const double guard_thr = 1e-280 * aT4;
      double sumR = 0.0, sumAbsFR = 0.0, SFRq = 0.0, SJq = 0.0;
      EdgeFn lo = planck_edge(P.nu[0] * beta);
      if (COUNT) flops += kFlopCellEval + lo.flops + (unsigned)(kFlopGroupEval * Nq);
      double Et_next = S.Erad[cell];
      for (int g = 0; g < Nq; ++g) {
        // a1: edge functions at the upper edge of group g
        const EdgeFn hi = planck_edge(P.nu[g + 1] * beta);
        if (COUNT) flops += hi.flops;
        const double Et = Et_next;
        if (g + 1 < Nq) Et_next = S.Erad[(long long)(g + 1) * stride + cell];
        // a2: group Planck integral and Doppler boundary terms (Eq. 11, 18, 22)
        const double Bt = aT4 * planck_dY(lo, hi);
        const double Db = aT4 * (hi.xi - lo.xi);
        const double D = aT4 * chis * fma(P.k_hi[g], hi.xi, -P.k_lo[g] * lo.xi);
        const double chiE = chis * P.k_mean[g];                  // = chi_B (alpha_Q = -1 for both)
        const double fourBmDb = fma(4.0, Bt, -Db);               // = 3 * denominator of Eq. 27 = T dBt/dT
        // a3: flux-mean opacity, Eq. 27, with the Wien-limit guard (S8)
        const double den = fourBmDb * (1.0 / 3.0);
        const double num = fma(chis * Bt, P.k_num[g], -D * (1.0 / 3.0));   // (chi_B+chi_E/3+alpha chi_E/3) Bt - D/3
        double chiF;
        if (!(den >= guard_thr) || isinf(den)) {
          chiF = chis * P.k_lo[g];
          if (evals == 0) cnt_guard++;
        } else if (den > 1e-290 && den < 1e290) {
          chiF = num * fast_rcp(den);
        } else {
          chiF = num / den;
        }
        if (!(fma(cdt, chiF, 1.0) > 0.0)) {
          if (evals == 0) cnt_den++;
          chiF = chiE;
        }
        // a4: residuals (Eq. 41; Eq. 42 solved for E_g)
        const double R = sm(SL_R, g);
        const double inv_chiE = inv_chis * P.inv_k_mean[g];
        const double itau = itau_c * P.inv_k_mean[g];
        const double W = P.onepa[g] * chiF * sm(SL_VF, g) * inv_c;
        const double Eg = fma(W * inv_chiE, inv_c, Bt) - R * itau;
        const double FR = Eg - Et - R;
        sumR += R;
        sumAbsFR += fabs(FR);
        // a5: Jacobian pieces (Eq. 44-47) folded into the arrowhead elimination (Eq. 48):
        //     1/J_gg = -q, q = 1/(1 + itau)
        const double q = fast_rcp(1.0 + itau);
        const double Jg0 = fourBmDb * dBscale;
        const double da = FR * q, db = Jg0 * q;
        SFRq += da;
        SJq += db;
        sm(SL_DA, g) = da;
        sm(SL_DB, g) = db;
        sm(SL_AG, g) = fma(chiE, Bt, -D * (1.0 / 3.0));          // chi_B Bt - D/3 (Eq. 51 source)
        sm(SL_CHIF, g) = chiF;
        lo = hi;
      }
      const double FG = Egs - Egas_t + c_over_chat * sumR;
      evals++;
      const double inv_Etot = 1.0 / Etot;
      if (fabs(FG) * inv_Etot < P.newton_tol && c_over_chat * sumAbsFR * inv_Etot < P.newton_tol) {
        phase = PH_FLUX;                                          // Eq. 49 met
      } else if (it >= P.newton_maxit) {
        cnt_newton_unconv++;
        phase = PH_FLUX;
      } else {
        // Newton step: eliminate the gas row
        //   dx0 = (-F_G + sum J0g F_R,g/Jgg) / (1 - sum J0g Jg0/Jgg),  dR_g = (F_R,g + Jg0 dx0) q
        const double dx0 = (-FG - c_over_chat * SFRq) / fma(c_over_chat, SJq, 1.0);
        double lam = 1.0;
        for (int h = 0; h < 10 && !((Egs + lam * dx0 - Ekin) * inv_Cv > 0.0); ++h) {
          lam *= 0.5;
          cnt_Tnonpos++;
        }
        Egs += lam * dx0;
        const double ldx = lam * dx0;
        for (int g = 0; g < Nq; ++g) sm(SL_R, g) = fma(lam, sm(SL_DA, g), fma(ldx, sm(SL_DB, g), sm(SL_R, g)));
        it++;
        if (COUNT) flops += kFlopStepCell + kFlopStepGroup * Nq;
      }
    }

    // ===== FLUX: energy commit (a6), closure + Eq. 51 (a7), Eq. 52 (a8), outer test (a9) =========
    if (phase == PH_FLUX) {
      const double inv_rho = 1.0 / rho;
      const double v0 = momk0 * inv_rho, v1 = momk1 * inv_rho, v2 = momk2 * inv_rho;
      double sumR = 0.0, dF0 = 0.0, dF1 = 0.0, dF2 = 0.0;
      bool rel_ok = true;
      for (int g = 0; g < Nq; ++g) {
        const long long o = (long long)g * stride + cell;
        const double Ft0 = S.Frad[0][o], Ft1 = S.Frad[1][o], Ft2 = S.Frad[2][o];
        const double Fk0 = fk(0, g), Fk1 = fk(1, g), Fk2 = fk(2, g);
        const double R = sm(SL_R, g);
        sumR += R;
        const double Enew = S.Erad[o] + R;                        // E_g^(t+1) = E_g^(t) + R_g
        double p0, p1, p2;
        closure_vP(P.closure, Enew, Fk0, Fk1, Fk2, v0, v1, v2, c, p0, p1, p2);
        const double w = P.onepa[g] * (chis * P.k_mean[g]);       // (1 + alpha) chi_E
        const double chiF = sm(SL_CHIF, g), A = sm(SL_AG, g);
        const double dn = fma(cdt, chiF, 1.0);                    // 1 + c_hat chi_F dt > 0 (guarded in EVAL)
        const double inv_dn = (dn > 1e-290 && dn < 1e290) ? fast_rcp(dn) : 1.0 / dn;
        const double Fn0 = fma(cdt, fma(v0, A, w * p0), Ft0) * inv_dn;
        const double Fn1 = fma(cdt, fma(v1, A, w * p1), Ft1) * inv_dn;
        const double Fn2 = fma(cdt, fma(v2, A, w * p2), Ft2) * inv_dn;
        dF0 += Fn0 - Ft0; dF1 += Fn1 - Ft1; dF2 += Fn2 - Ft2;
        if (P.outer_stop == 1) {
          const double e0 = Fn0 - Fk0, e1 = Fn1 - Fk1, e2 = Fn2 - Fk2;
          const double d2 = fma(e0, e0, fma(e1, e1, e2 * e2));
          const double f2 = fma(Fn0, Fn0, fma(Fn1, Fn1, Fn2 * Fn2));
          // |dF| <= rel |F|  (compared squared unless the squares leave the normal range)
          bool ok;
          if (f2 > 1e-280 && f2 < 1e280) ok = d2 <= P.outer_rel_tol * P.outer_rel_tol * f2;
          else ok = norm3(e0, e1, e2) <= P.outer_rel_tol * norm3(Fn0, Fn1, Fn2);
          if (!ok) rel_ok = false;
        }
        fk(0, g) = Fn0; fk(1, g) = Fn1; fk(2, g) = Fn2;
      }
      Egas_new = Egas_t - c_over_chat * sumR;
      momn0 = momt0 - dF0 * icc; momn1 = momt1 - dF1 * icc; momn2 = momt2 - dF2 * icc;   // Eq. 52
      trips++;
      if (COUNT) flops += kFlopOuterCell + kFlopOuterGroup * Nq;

      const double vn0 = momn0 * inv_rho, vn1 = momn1 * inv_rho, vn2 = momn2 * inv_rho;
      double dW = 0.0, sumAbsR = 0.0;
      for (int g = 0; g < Nq; ++g) {
        const double vFn = fma(vn0, fk(0, g), fma(vn1, fk(1, g), vn2 * fk(2, g)));
        const double wf = P.onepa[g] * sm(SL_CHIF, g) * inv_c;
        dW += fabs(wf * (vFn - sm(SL_VF, g)));
        sumAbsR += fabs(sm(SL_R, g));
        sm(SL_VF, g) = vFn;                                       // lagged v.F_g of the next trip
      }
      if (P.outer_stop == 1) {
        const double d = norm3(momn0 - momk0, momn1 - momk1, momn2 - momk2);
        if (!(d <= P.outer_rel_tol * norm3(momn0, momn1, momn2))) rel_ok = false;
      }
      const double delta = dW * (chat / c) * dt;
      if (delta <= P.outer_tol * fmax(sumAbsR, Etot) && rel_ok) {
        phase = PH_STORE;
      } else if (k == P.outer_maxit - 1) {
        cnt_outer_unconv++;
        phase = PH_STORE;
      } else {
        momk0 = momn0; momk1 = momn1; momk2 = momn2;
        Ekin = (momk0 * momk0 + momk1 * momk1 + momk2 * momk2) / (2.0 * rho);
        k++;
        it = 0;
        if ((Egs - Ekin) * inv_Cv > 0.0) phase = PH_EVAL;
        else { cnt_Tnonpos++; phase = PH_STORE; }
      }
    }

    // ===== STORE (a10) ============================================================================
    if (phase == PH_STORE) {
      if (trips > 0) {
        S.mom[0][cell] = momn0; S.mom[1][cell] = momn1; S.mom[2][cell] = momn2;
        S.Egas[cell] = Egas_new;   // total gas energy; E_int = Egas - |mom|^2/(2 rho)
        for (int g = 0; g < Nq; ++g) {
          const long long o = (long long)g * stride + cell;
          S.Erad[o] = S.Erad[o] + sm(SL_R, g);
          S.Frad[0][o] = fk(0, g);
          S.Frad[1][o] = fk(1, g);
          S.Frad[2][o] = fk(2, g);
        }
      }
      cnt_evals += evals;
      cnt_trips += trips;
      cnt_cells++;
      atomicAdd(&s_hist[evals < MGRHD_HIST ? evals : MGRHD_HIST - 1], 1u);
      atomicAdd(&s_hist[MGRHD_HIST + (trips < MGRHD_HIST ? trips : MGRHD_HIST - 1)], 1u);
      phase = PH_LOAD;
    }
  }

  // ---- diagnostics: warp-reduce the scalar counters, one atomic per warp ------------------
  unsigned int vals[8] = {cnt_cells, cnt_newton_unconv, cnt_outer_unconv, cnt_Tnonpos,
                          cnt_guard, cnt_den, cnt_evals, cnt_trips};
#pragma unroll
  for (int s = 0; s < 8; ++s) {
    unsigned int v = vals[s];
    for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(FULL, v, off);
    if (lane == 0 && v) atomicAdd(&stats[s], (unsigned long long)v);
  }
  if (COUNT) {
    for (int off = 16; off > 0; off >>= 1) flops += __shfl_xor_sync(FULL, flops, off);
    if (lane == 0) atomicAdd(&stats[kStatFlops], flops);
  }
  __syncthreads();
  for (int t = threadIdx.x; t < 2 * MGRHD_HIST; t += THREADS)
    if (s_hist[t]) atomicAdd(&stats[kStatNewtonHist + t], (unsigned long long)s_hist[t]);
}

// Per-cell conserved totals: E_gas + (c/c_hat) sum E_g and
// rho v + (c c_hat)^-1 sum F_g.
__global__ void conserved_totals_kernel(const __grid_constant__ StatePtrs S, int Nq, long long n,
                                        long long stride, double c, double chat,
                                        double* __restrict__ outE, double* __restrict__ outP) {
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n;
       i += (long long)gridDim.x * blockDim.x) {
    double sE = 0.0, s0 = 0.0, s1 = 0.0, s2 = 0.0;
    for (int g = 0; g < Nq; ++g) {
      const long long o = (long long)g * stride + i;
      sE += S.Erad[o];
      s0 += S.Frad[0][o]; s1 += S.Frad[1][o]; s2 += S.Frad[2][o];
    }
    const double icc = 1.0 / (c * chat);
    outE[i] = S.Egas[i] + (c / chat) * sE;
    outP[i] = S.mom[0][i] + icc * s0;
    outP[n + i] = S.mom[1][i] + icc * s1;
    outP[2 * n + i] = S.mom[2][i] + icc * s2;
  }
}

// Diagnostic: the edge functions on an array of x (tests pin them against the oracle's).
__global__ void planck_edge_kernel(const double* __restrict__ x, long long n, double* __restrict__ yz,
                                   double* __restrict__ xi, int* __restrict__ is_y) {
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n;
       i += (long long)gridDim.x * blockDim.x) {
    const EdgeFn e = planck_edge(x[i]);
    yz[i] = e.yz;
    xi[i] = e.xi;
    is_y[i] = e.small ? 1 : 0;
  }
}

// Dependency-free DFMA throughput probe: 8 independent chains per thread.
__global__ void dfma_peak_kernel(long long iters, double* out) {
  double a0 = threadIdx.x * 1e-9, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5,
         a6 = a0 + 6, a7 = a0 + 7;
  const double m = 0.999999, b = 1e-7;
  for (long long k = 0; k < iters; k += 8) {
    a0 = fma(a0, m, b); a1 = fma(a1, m, b); a2 = fma(a2, m, b); a3 = fma(a3, m, b);
    a4 = fma(a4, m, b); a5 = fma(a5, m, b); a6 = fma(a6, m, b); a7 = fma(a7, m, b);
  }
  const double s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
  if (s == 123.456) out[0] = s;  // never true; keeps the chains alive
}

}  // namespace mgrhd
