// mgrhd_api.cu -- host side of the C ABI declared in include/mgrhd.h: argument checks,
// table generation, launches, the slab-pipelined host-buffer path and diagnostics.
// Product code; shares nothing with oracle/.  No CPU fallback anywhere: every computing
// entry point launches the CUDA kernels of mgrhd_kernels.cuh or fails.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>

#include "mgrhd_general.cuh"
#include "mgrhd_transport.cuh"

using namespace mgrhd;

namespace {

thread_local char g_err[512] = "";

bool cuda_ok(cudaError_t e, const char* what) {
  if (e == cudaSuccess) return true;
  std::snprintf(g_err, sizeof g_err, "%s: %s", what, cudaGetErrorString(e));
  return false;
}
#define CU(call) do { if (!cuda_ok((call), #call)) return MGRHD_ERR_CUDA; } while (0)

// zeta(2n) for n >= 1 in long double: direct sum + Euler-Maclaurin tail.
long double zeta_even(int n) {
  const long double PI = 3.14159265358979323846264338327950288L;
  if (n == 1) return PI * PI / 6.0L;
  if (n == 2) return PI * PI * PI * PI / 90.0L;
  const int s = 2 * n, M = 64;
  long double sum = 0.0L;
  for (int k = M - 1; k >= 1; --k) sum += powl((long double)k, -(long double)s);
  const long double m = (long double)M;
  // tail: int_M^inf x^-s dx + M^-s/2 + s M^(-s-1)/12 - s(s+1)(s+2) M^(-s-3)/720
  sum += powl(m, 1.0L - s) / (s - 1.0L) + 0.5L * powl(m, -(long double)s) +
         s * powl(m, -s - 1.0L) / 12.0L - s * (s + 1.0L) * (s + 2.0L) * powl(m, -s - 3.0L) / 720.0L;
  return sum;
}

// b_{2n} = B_{2n}/(2n)! = (-1)^(n+1) 2 zeta(2n)/(2 pi)^(2n): Maclaurin coefficients of
// t/(e^t-1) = 1 - t/2 + sum_n b_{2n} t^(2n).
long double bern_over_fact(int n) {
  const long double TWO_PI = 6.28318530717958647692528676655900577L;
  long double b = 2.0L * zeta_even(n) / powl(TWO_PI, 2.0L * n);
  return (n % 2 == 0) ? -b : b;
}

const long double kC15Pi4L = 15.0L / (3.14159265358979323846264338327950288L * 3.14159265358979323846264338327950288L *
                                      3.14159265358979323846264338327950288L * 3.14159265358979323846264338327950288L);

// Reference values for the mid-range fits, long double, x >= 1:
//   Z(x) = C sum_n e^{-nx}(x^3/n + 3x^2/n^2 + 6x/n^3 + 6/n^4),  Xi(x) = C x^4/(e^x - 1).
long double Z_host(long double x) {
  long double sum = 0.0L;
  for (int n = 1; n <= 200; ++n) {
    const long double q = 1.0L / n;
    const long double term = expl(-n * x) * q * (x * x * x + q * (3.0L * x * x + q * (6.0L * x + q * 6.0L)));
    sum += term;
    if (term < 1e-24L * sum) break;
  }
  return kC15Pi4L * sum;
}
long double Xi_host(long double x) { return kC15Pi4L * x * x * x * x / expm1l(x); }

// Chebyshev interpolation of f on [a,b] with N nodes, truncated to M terms and rewritten as a
// monomial series in t = (2x - a - b)/(b - a): out[k] t^k.
void cheb_fit_monomial(long double (*f)(long double), long double a, long double b, int N, int M, double* out) {
  const long double PI = 3.14159265358979323846264338327950288L;
  long double fx[64], ck[64], mono[64] = {0}, Tkm1[64] = {0}, Tk[64] = {0}, Tn[64];
  for (int j = 0; j < N; ++j) fx[j] = f(0.5L * (a + b) + 0.5L * (b - a) * cosl(PI * (j + 0.5L) / N));
  for (int k = 0; k < M; ++k) {
    long double s = 0.0L;
    for (int j = 0; j < N; ++j) s += fx[j] * cosl(PI * k * (j + 0.5L) / N);
    ck[k] = 2.0L * s / N;
  }
  ck[0] *= 0.5L;
  // T_0 = 1, T_1 = t, T_{k+1} = 2 t T_k - T_{k-1}, as monomial coefficient vectors
  Tkm1[0] = 1.0L;
  Tk[1] = 1.0L;
  mono[0] += ck[0];
  if (M > 1) mono[1] += ck[1];
  for (int k = 2; k < M; ++k) {
    for (int i = 0; i < 64; ++i) Tn[i] = -Tkm1[i];
    for (int i = 0; i + 1 < 64; ++i) Tn[i + 1] += 2.0L * Tk[i];
    for (int i = 0; i < 64; ++i) { mono[i] += ck[k] * Tn[i]; Tkm1[i] = Tk[i]; Tk[i] = Tn[i]; }
  }
  for (int k = 0; k < M; ++k) out[k] = (double)mono[k];
}

void fill_planck_tables(PlanckTables& t) {
  for (int n = 1; n <= kSmallTerms; ++n) {
    const long double b = bern_over_fact(n);
    t.sp[n - 1].a = (double)(b / (2.0L * n + 3.0L));
    t.sp[n - 1].b = (double)b;
  }
  double mz[kMidTerms], mx[kMidTerms];
  cheb_fit_monomial(Z_host, kXS, kXL, 48, kMidTerms, mz);
  cheb_fit_monomial(Xi_host, kXS, kXL, 48, kMidTerms, mx);
  for (int k = 0; k < kMidTerms; ++k) { t.mp[k].a = mz[k]; t.mp[k].b = mx[k]; }
  t.mid_s = (double)(2.0L / ((long double)kXL - (long double)kXS));
  t.mid_o = (double)(-((long double)kXL + (long double)kXS) / ((long double)kXL - (long double)kXS));
  for (int n = 1; n <= kLargeTerms; ++n) {
    const long double q = 1.0L / n;
    t.l32[n - 1].a = (double)(kC15Pi4L * q);
    t.l32[n - 1].b = (double)(3.0L * kC15Pi4L * q * q);
    t.l10[n - 1].a = (double)(6.0L * kC15Pi4L * q * q * q);
    t.l10[n - 1].b = (double)(6.0L * kC15Pi4L * q * q * q * q);
  }
}

// Reference functions of the per-interval rows, long double.
//   x < 1:  Y/(x^3) = C (1/3 - x/8 + sum b_2n x^2n/(2n+3)),  Xi/x^3 = C x/(e^x - 1)
//   x >= 8: Z e^x, Xi e^x = C x^4/(1 - e^-x)
long double Yx3_host(long double x) {
  long double s = 1.0L / 3.0L - x / 8.0L, p = 1.0L;
  for (int n = 1; n <= 30; ++n) {
    p *= x * x;
    s += bern_over_fact(n) * p / (2.0L * n + 3.0L);
  }
  return kC15Pi4L * s;
}
long double Xix3_host(long double x) { return x == 0.0L ? kC15Pi4L : kC15Pi4L * x / expm1l(x); }
long double Zex_host(long double x) { return Z_host(x) * expl(x); }
long double Xiex_host(long double x) { return kC15Pi4L * x * x * x * x / (-expm1l(-x)); }

// rows[kRows * kRowStride], layout in mgrhd_params.h
void fill_planck_rows(double* rows) {
  for (int j = 0; j < kRows; ++j) {
    double* r = rows + j * kRowStride;
    long double a, b;
    if (j == 0) { a = 0.0L; b = 0.5L; }
    else {
      const int bin = (j - 1) / 8, m = (j - 1) % 8;
      const long double lo = ldexpl(0.5L, bin), w = lo / 8.0L;
      a = lo + m * w; b = a + w;
    }
    double cy[kRowTerms], cx[kRowTerms];
    if (j == kRows - 1) {                       // x >= 64: e^-x < 2e-28, Z e^x and Xi e^x are polynomials in x
      for (int k = 0; k < kRowTerms; ++k) { cy[k] = 0.0; cx[k] = 0.0; }
      cy[0] = (double)(6.0L * kC15Pi4L); cy[1] = cy[0]; cy[2] = (double)(3.0L * kC15Pi4L); cy[3] = (double)kC15Pi4L;
      cx[4] = (double)kC15Pi4L;
      r[0] = 0.0; r[1] = 1.0;
    } else {
      long double (*fy)(long double) = b <= 1.0L ? Yx3_host : (b <= 8.0L ? Z_host : Zex_host);
      long double (*fx)(long double) = b <= 1.0L ? Xix3_host : (b <= 8.0L ? Xi_host : Xiex_host);
      cheb_fit_monomial(fy, a, b, 32, kRowTerms, cy);
      cheb_fit_monomial(fx, a, b, 32, kRowTerms, cx);
      r[0] = (double)(0.5L * (a + b)); r[1] = (double)(2.0L / (b - a));
    }
    for (int k = 0; k < kRowTerms; ++k) { r[2 + 2 * k] = cy[k]; r[3 + 2 * k] = cx[k]; }
  }
}

std::once_flag g_tables_once[16];  // per device
cudaError_t g_tables_err[16];

// The host copy of the tables: filled once per process under its own flag (two threads may
// initialise contexts on different devices at the same time), read-only afterwards.
const PlanckTables* host_planck_tables() {
  static PlanckTables t[2];
  static std::once_flag once;
  std::call_once(once, []() {
    fill_planck_tables(t[0]);
    t[1] = t[0];
  });
  return t;
}
const double* host_planck_rows() {
  static double rows[kRows * kRowStride];
  static std::once_flag once;
  std::call_once(once, []() { fill_planck_rows(rows); });
  return rows;
}

cudaError_t upload_tables_for_current_device() {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= 16) return cudaErrorInvalidDevice;
  const PlanckTables* t = host_planck_tables();
  const double* rows = host_planck_rows();
  std::call_once(g_tables_once[dev], [dev, t, rows]() {
    g_tables_err[dev] = cudaMemcpyToSymbol(mgrhd_c_planck, t, 2 * sizeof(PlanckTables));
    if (g_tables_err[dev] == cudaSuccess)
      g_tables_err[dev] = cudaMemcpyToSymbol(mgrhd_g_rows, rows, kRows * kRowStride * sizeof(double));
  });
  return g_tables_err[dev];
}

constexpr int kSlabs = 3;                       // host path: slabs in flight
constexpr long long kSlabBytes = 512ll << 20;   // largest slab (measured at 256^3 x 32, 3 slabs: 96 MB 444 ms, 256 MB 422,
                                                // 512 MB 410, 768 MB 405, 1 GB unstable; 4 or more slabs, or smaller ones, are slower)

}  // namespace

struct mgrhd_ctx {
  Params P;
  GenParams G;
  int general;                        // 1: the general kernel (free-slope spectrum, opacity_kind 2) runs
  double* d_lnk;                      // opacity_kind 2: device copy of the edge table
  int device;
  int sm_count;
  unsigned long long* d_stats;
  cudaStream_t last_stream;
  long long launches;
  int count_flops;
  int cfg_l;
  int cfg_nq, cfg_threads, cfg_bps;   // kernel instantiation, CTA size, resident CTAs per SM
  double* scratch;                    // lagged-flux scratch of the device path
  double* slab_scratch[kSlabs];       // ... and of each host-path slab stream
  // host-buffer path scratch (lazily allocated)
  double* slab[kSlabs];
  long long slab_cells;
  cudaStream_t slab_stream[kSlabs];
};

// One instantiation per (lanes per cell L, steps per lane NQL, CTA size): chosen so that the
// [slot][step][thread] state fits in shared memory (SL_COUNT * NQL * THREADS * 8 bytes <= 227 KB)
// with as many threads per SM as the register file allows.
template <int L, int NQL, int THREADS, bool KT>
struct Inst {
  template <bool SRC, bool COUNT>
  static auto kernel() { return source_update_kernel<L, NQL, THREADS, KT, SRC, COUNT>; }
  static constexpr size_t kSmem = (size_t)SL_COUNT * NQL * THREADS * sizeof(double);
  static cudaError_t configure(int* blocks_per_sm) {
    cudaError_t e = cudaSuccess;
    const void* k[4] = {(const void*)kernel<false, false>(), (const void*)kernel<false, true>(),
                        (const void*)kernel<true, false>(), (const void*)kernel<true, true>()};
    for (int i = 0; i < 4 && e == cudaSuccess; ++i)
      e = cudaFuncSetAttribute(k[i], cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmem);
    if (e == cudaSuccess)
      e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks_per_sm, kernel<false, false>(), THREADS, kSmem);
    return e;
  }
  static void launch(bool count, unsigned blocks, cudaStream_t st, const Params& P, const StatePtrs& S,
                     unsigned long long* stats, double* scratch) {
    const bool src = S.Srad != nullptr;
    if (src && count) kernel<true, true>()<<<blocks, THREADS, kSmem, st>>>(P, S, stats, scratch);
    else if (src) kernel<true, false>()<<<blocks, THREADS, kSmem, st>>>(P, S, stats, scratch);
    else if (count) kernel<false, true>()<<<blocks, THREADS, kSmem, st>>>(P, S, stats, scratch);
    else kernel<false, false>()<<<blocks, THREADS, kSmem, st>>>(P, S, stats, scratch);
  }
};

// WHAT(L, NQL, THREADS): lanes per cell, steps per lane (L*NQL >= Nq), CTA size -- measured best
// on B200 for each bracket of Nq.
#define MGRHD_DISPATCH(Nq, WHAT)                               \
  do {                                                         \
    if ((Nq) <= 4) { WHAT(1, 4, 256); }                        \
    else if ((Nq) <= 8) { WHAT(1, 8, 384); }                   \
    else if ((Nq) <= 16) { WHAT(2, 8, 384); }                  \
    else if ((Nq) <= 32) { WHAT(4, 8, 384); }                  \
    else { WHAT(4, 16, 256); }                                 \
  } while (0)

// Fills ctx->cfg_* for ctx->P.Nq (called once by mgrhd_init).
static cudaError_t configure_ctx(mgrhd_ctx* ctx) {
  cudaError_t e = cudaSuccess;
#define MGRHD_CFG(LL, Q, T)                                                                                 \
  e = kt ? Inst<LL, Q, T, true>::configure(&ctx->cfg_bps) : Inst<LL, Q, T, false>::configure(&ctx->cfg_bps); \
  ctx->cfg_l = LL; ctx->cfg_nq = Q; ctx->cfg_threads = T
  const bool kt = ctx->G.opacity_kind == 1;
  MGRHD_DISPATCH(ctx->P.Nq, MGRHD_CFG);
#undef MGRHD_CFG
  if (e == cudaSuccess && ctx->cfg_bps < 1) e = cudaErrorLaunchOutOfResources;
  return e;
}

// Bytes of scratch one launch needs at most: the head (work counter) and 3 * NQL doubles per resident thread.
static size_t scratch_bytes(const mgrhd_ctx* ctx) {
  return kScratchHead * sizeof(double) + (size_t)3 * ctx->cfg_nq * sizeof(double) * (size_t)ctx->sm_count * ctx->cfg_bps * ctx->cfg_threads;
}

extern "C" {

const char* mgrhd_last_error(void) { return g_err; }

int mgrhd_init(mgrhd_ctx** out, const double* edges, int Nq, const mgrhd_units* u,
               const mgrhd_opacity_model* m) {
  if (out) *out = nullptr;
  if (!out || !edges || !u || !m) return MGRHD_ERR_ARG;
  if (m->opacity_kind < 0 || m->opacity_kind > 2 || m->outer_mode < 0 || m->outer_mode > 1) return MGRHD_ERR_ARG;
  const bool tab = m->opacity_kind == 2;
  if (!tab && (!m->kappa_lo || !m->alpha)) return MGRHD_ERR_ARG;
  if (tab && (!m->lnk_edge || m->NT < 1)) return MGRHD_ERR_ARG;
  if (Nq < 1 || Nq > MGRHD_MAX_GROUPS) return MGRHD_ERR_ARG;
  if (m->closure < 0 || m->closure > 1 || m->spectrum < 0 || m->spectrum > 1) return MGRHD_ERR_ARG;
  if (m->outer_stop < 0 || m->outer_stop > 1 || m->newton_maxit < 1 || m->outer_maxit < 1)
    return MGRHD_ERR_ARG;
  if (!(u->a_rad > 0) || !(u->k_B > 0) || !(u->h_planck > 0) || !(u->mean_mass > 0) ||
      !(u->gamma > 1) || !(m->newton_tol > 0) || !(m->outer_tol > 0))
    return MGRHD_ERR_RANGE;
  if (m->opacity_kind == 1 && (!(m->T_ref > 0) || !std::isfinite(m->T_ref) || !std::isfinite(m->p_T))) return MGRHD_ERR_RANGE;
  if (tab && m->NT > 1 && (!(m->dlnT > 0) || !std::isfinite(m->dlnT) || !std::isfinite(m->lnT0))) return MGRHD_ERR_RANGE;
  if (tab)
    for (long long i = 0; i < (long long)(Nq + 1) * m->NT; ++i)
      if (!std::isfinite(m->lnk_edge[i])) return MGRHD_ERR_RANGE;
  for (int g = 0; g < Nq; ++g) {
    if (!(edges[g] >= 0.0) || !(edges[g + 1] > edges[g])) return MGRHD_ERR_EDGES;
    const bool open_group = edges[g] == 0.0 || std::isinf(edges[g + 1]);
    if (tab) {
      if (open_group) return MGRHD_ERR_ALPHA;       // Eq. 20 needs both edge values of every group
      continue;
    }
    if (m->alpha[g] != 0.0 && open_group) return MGRHD_ERR_ALPHA;
    // kappa = 0 makes Eq. 42 singular (E_g = ... /chi_E): rejected, as are inf/NaN
    if (!std::isfinite(m->alpha[g]) || !(m->kappa_lo[g] > 0.0) || !std::isfinite(m->kappa_lo[g])) return MGRHD_ERR_RANGE;
  }
  mgrhd_ctx* ctx = new (std::nothrow) mgrhd_ctx();
  if (!ctx) return MGRHD_ERR_ARG;
  std::memset(ctx, 0, sizeof *ctx);
  Params& P = ctx->P;
  P.Nq = Nq;
  P.closure = m->closure;
  P.newton_maxit = m->newton_maxit;
  P.outer_maxit = m->outer_maxit;
  P.outer_stop = m->outer_stop;
  P.newton_tol = m->newton_tol;
  P.outer_tol = m->outer_tol;
  P.outer_rel_tol = m->outer_rel_tol;
  P.a_rad = u->a_rad;
  P.h_over_k = u->h_planck / u->k_B;
  P.cv_over_rho = u->k_B / ((u->gamma - 1.0) * u->mean_mass);
  for (int g = 0; g <= Nq; ++g) P.nu[g] = edges[g];
  P.inv_T_ref = m->opacity_kind == 1 ? 1.0 / m->T_ref : 1.0;
  P.p_T = m->opacity_kind == 1 ? m->p_T : 0.0;
  GenParams& G = ctx->G;
  G.spectrum = m->spectrum;
  G.opacity_kind = m->opacity_kind;
  G.outer_mode = m->outer_mode;
  G.NT = tab ? m->NT : 0;
  G.lnT0 = tab ? m->lnT0 : 0.0;
  G.inv_dlnT = tab && m->NT > 1 ? 1.0 / m->dlnT : 0.0;
  for (int g = 0; g < Nq; ++g) {
    const bool open_group = edges[g] == 0.0 || std::isinf(edges[g + 1]);
    G.lnr[g] = open_group ? 0.0 : std::log(edges[g + 1] / edges[g]);
    G.width[g] = edges[g + 1] - edges[g];
    G.inv_lnnb[g] = 0.0;
    if (g + 1 < Nq && edges[g] > 0.0 && std::isfinite(edges[g + 2]))     // Eq. A1 between groups g and g + 1
      G.inv_lnnb[g] = 1.0 / std::log(std::sqrt(edges[g + 2] * edges[g + 1]) / std::sqrt(edges[g + 1] * edges[g]));
  }
  ctx->general = (m->spectrum == 1 || tab || m->outer_mode == 1) ? 1 : 0;
  for (int g = 0; g < Nq; ++g) {
    const double a = tab ? 0.0 : m->alpha[g], k = tab ? 1.0 : m->kappa_lo[g];
    P.alpha[g] = a;
    P.k_lo[g] = k;
    if (a == 0.0) {                       // piecewise constant, Eq. 17
      P.k_hi[g] = k;
      P.k_mean[g] = k;
    } else {                              // Eq. 19 at nu_g+; Eq. 30 with alpha_Q = -1
      const double z = a * std::log(edges[g + 1] / edges[g]);
      P.k_hi[g] = k * std::exp(z);
      P.k_mean[g] = k * (std::expm1(z) / z);
    }
    P.inv_k_mean[g] = 1.0 / P.k_mean[g];
    P.k_num[g] = P.k_mean[g] * ((4.0 + a) / 3.0);
    P.onepa[g] = 1.0 + a;
  }
  cudaError_t e = cudaGetDevice(&ctx->device);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, ctx->device);
  if (e == cudaSuccess) e = upload_tables_for_current_device();
  if (e == cudaSuccess) e = configure_ctx(ctx);
  if (e == cudaSuccess) e = cudaMalloc(&ctx->scratch, scratch_bytes(ctx));
  if (e == cudaSuccess && tab) {
    const size_t bytes = (size_t)(Nq + 1) * m->NT * sizeof(double);
    e = cudaMalloc(&ctx->d_lnk, bytes);
    if (e == cudaSuccess) e = cudaMemcpy(ctx->d_lnk, m->lnk_edge, bytes, cudaMemcpyHostToDevice);
    G.lnk_edge = ctx->d_lnk;
  }
  if (e == cudaSuccess) e = cudaMalloc(&ctx->d_stats, kStatCount * sizeof(unsigned long long));
  if (e == cudaSuccess) e = cudaMemset(ctx->d_stats, 0, kStatCount * sizeof(unsigned long long));
  if (e != cudaSuccess) {
    cuda_ok(e, "mgrhd_init");
    if (ctx->d_stats) cudaFree(ctx->d_stats);
    if (ctx->scratch) cudaFree(ctx->scratch);
    if (ctx->d_lnk) cudaFree(ctx->d_lnk);
    delete ctx;
    return MGRHD_ERR_CUDA;
  }
  *out = ctx;
  return MGRHD_OK;
}

static int check_call(const mgrhd_ctx* ctx, const mgrhd_state* s, long long n, double dt, double c,
                      double chat) {
  if (!ctx || !s || n < 0) return MGRHD_ERR_ARG;
  int dev = -1;                      // a context belongs to the device that was current in mgrhd_init
  if (cudaGetDevice(&dev) != cudaSuccess || dev != ctx->device) return MGRHD_ERR_ARG;
  if (!(dt > 0.0) || !(c > 0.0) || !(chat > 0.0) || chat > c) return MGRHD_ERR_RANGE;
  if (n > 0 && (!s->rho || !s->mom[0] || !s->mom[1] || !s->mom[2] || !s->Egas || !s->Erad ||
                !s->Frad[0] || !s->Frad[1] || !s->Frad[2]))
    return MGRHD_ERR_ARG;
  return MGRHD_OK;
}

static int launch_update(mgrhd_ctx* ctx, const StatePtrs& S, long long n, long long stride, double dt,
                         double c, double chat, cudaStream_t st, double* scratch) {
  Params P = ctx->P;
  P.dt = dt; P.c = c; P.c_hat = chat; P.ncells = n; P.stride = stride;
  // persistent grid: one CTA per resident slot, fewer when the problem is small
  long long blocks = (long long)ctx->sm_count * ctx->cfg_bps;
  const long long cells_per_cta = ctx->cfg_threads / ctx->cfg_l;
  const long long want = (n + cells_per_cta - 1) / cells_per_cta;
  if (blocks > want) blocks = want;
  const bool count = ctx->count_flops != 0;
  CU(cudaMemsetAsync(scratch, 0, kScratchHead * sizeof(double), st));   // work counter of the chunk scheduler
  if (ctx->general) {
    // one warp per cell, 8 warps per CTA, persistent grid (8 CTAs per SM at most)
    long long gb = (n + 7) / 8;
    const long long cap = (long long)ctx->sm_count * 8;
    if (gb > cap) gb = cap;
    if (P.Nq <= 32) {
      if (count) source_update_general_kernel<1, true><<<(unsigned)gb, 256, 0, st>>>(P, ctx->G, S, ctx->d_stats);
      else source_update_general_kernel<1, false><<<(unsigned)gb, 256, 0, st>>>(P, ctx->G, S, ctx->d_stats);
    } else {
      if (count) source_update_general_kernel<2, true><<<(unsigned)gb, 256, 0, st>>>(P, ctx->G, S, ctx->d_stats);
      else source_update_general_kernel<2, false><<<(unsigned)gb, 256, 0, st>>>(P, ctx->G, S, ctx->d_stats);
    }
    ctx->launches++;
    ctx->last_stream = st;
    CU(cudaGetLastError());
    return MGRHD_OK;
  }
  const bool kt = ctx->G.opacity_kind == 1;
#define MGRHD_GO(LL, Q, T)                                                                        \
  if (kt) Inst<LL, Q, T, true>::launch(count, (unsigned)blocks, st, P, S, ctx->d_stats, scratch); \
  else Inst<LL, Q, T, false>::launch(count, (unsigned)blocks, st, P, S, ctx->d_stats, scratch)
  MGRHD_DISPATCH(P.Nq, MGRHD_GO);
#undef MGRHD_GO
  ctx->launches++;
  ctx->last_stream = st;
  CU(cudaGetLastError());
  return MGRHD_OK;
}

static StatePtrs to_ptrs(const mgrhd_state* s) {
  StatePtrs S;
  S.rho = s->rho;
  for (int i = 0; i < 3; ++i) { S.mom[i] = s->mom[i]; S.Frad[i] = s->Frad[i]; }
  S.Egas = s->Egas;
  S.Erad = s->Erad;
  S.kappa_scale = s->kappa_scale;
  S.Srad = s->Srad;
  return S;
}

int mgrhd_source_update(mgrhd_ctx* ctx, const mgrhd_state* s, long long n, double dt, double c,
                        double chat, void* stream) {
  int rc = check_call(ctx, s, n, dt, c, chat);
  if (rc != MGRHD_OK) return rc;
  if (n == 0) return MGRHD_OK;
  return launch_update(ctx, to_ptrs(s), n, n, dt, c, chat, (cudaStream_t)stream, ctx->scratch);
}

int mgrhd_conserved_totals(mgrhd_ctx* ctx, const mgrhd_state* s, long long n, double c, double chat,
                           double* outE, double* outP, void* stream) {
  int rc = check_call(ctx, s, n, 1.0, c, chat);
  if (rc != MGRHD_OK) return rc;
  if (!outE || !outP) return MGRHD_ERR_ARG;
  if (n == 0) return MGRHD_OK;
  long long blocks = (n + 255) / 256;
  const long long cap = (long long)ctx->sm_count * 32;
  if (blocks > cap) blocks = cap;
  conserved_totals_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(
      to_ptrs(s), ctx->P.Nq, n, n, c, chat, outE, outP);
  ctx->launches++;
  ctx->last_stream = (cudaStream_t)stream;
  CU(cudaGetLastError());
  return MGRHD_OK;
}

int mgrhd_source_update_host(mgrhd_ctx* ctx, const mgrhd_state* s, long long n, double dt, double c,
                             double chat) {
  int rc = check_call(ctx, s, n, dt, c, chat);
  if (rc != MGRHD_OK) return rc;
  if (n == 0) return MGRHD_OK;
  const int Nq = ctx->P.Nq;
  const long long per_cell = 6 + 5ll * Nq;     // rho, mom[3], Egas, kappa_scale, Erad, Frad[3], Srad
  {
    // slab size: a third of the cells (so that three slabs are in flight), at most kSlabBytes; grown when a larger call comes
    long long sc = kSlabBytes / (8 * per_cell);
    const long long third = (n + kSlabs - 1) / kSlabs;
    if (sc > third) sc = third;
    sc = ((sc + 1023) / 1024) * 1024;
    if (!ctx->slab[0] || sc > ctx->slab_cells) {
      for (int j = 0; j < kSlabs; ++j) {
        if (ctx->slab[j]) { CU(cudaStreamSynchronize(ctx->slab_stream[j])); CU(cudaFree(ctx->slab[j])); ctx->slab[j] = nullptr; }
        CU(cudaMalloc(&ctx->slab[j], (size_t)sc * per_cell * sizeof(double)));
        if (!ctx->slab_scratch[j]) CU(cudaMalloc(&ctx->slab_scratch[j], scratch_bytes(ctx)));
        if (!ctx->slab_stream[j]) CU(cudaStreamCreateWithFlags(&ctx->slab_stream[j], cudaStreamNonBlocking));
      }
      ctx->slab_cells = sc;
    }
  }
  const long long sc = ctx->slab_cells;
  const size_t pitch_h = (size_t)n * sizeof(double), pitch_d = (size_t)sc * sizeof(double);
  int j = 0;
  for (long long lo = 0; lo < n; lo += sc, j = (j + 1) % kSlabs) {
    const long long m = (n - lo < sc) ? (n - lo) : sc;
    const size_t w = (size_t)m * sizeof(double);
    cudaStream_t st = ctx->slab_stream[j];
    double* d = ctx->slab[j];
    StatePtrs S;
    double* q = d;
    S.rho = q; q += sc;
    for (int i = 0; i < 3; ++i) { S.mom[i] = q; q += sc; }
    S.Egas = q; q += sc;
    double* d_ks = q; q += sc;
    S.kappa_scale = s->kappa_scale ? d_ks : nullptr;
    S.Erad = q; q += sc * Nq;
    for (int i = 0; i < 3; ++i) { S.Frad[i] = q; q += sc * Nq; }
    double* d_S = q; q += sc * Nq;
    S.Srad = s->Srad ? d_S : nullptr;
    // host -> device
    CU(cudaMemcpyAsync((void*)S.rho, s->rho + lo, w, cudaMemcpyHostToDevice, st));
    for (int i = 0; i < 3; ++i) CU(cudaMemcpyAsync(S.mom[i], s->mom[i] + lo, w, cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(S.Egas, s->Egas + lo, w, cudaMemcpyHostToDevice, st));
    if (s->kappa_scale) CU(cudaMemcpyAsync(d_ks, s->kappa_scale + lo, w, cudaMemcpyHostToDevice, st));
    CU(cudaMemcpy2DAsync(S.Erad, pitch_d, s->Erad + lo, pitch_h, w, Nq, cudaMemcpyHostToDevice, st));
    for (int i = 0; i < 3; ++i)
      CU(cudaMemcpy2DAsync(S.Frad[i], pitch_d, s->Frad[i] + lo, pitch_h, w, Nq, cudaMemcpyHostToDevice, st));
    if (s->Srad) CU(cudaMemcpy2DAsync(d_S, pitch_d, s->Srad + lo, pitch_h, w, Nq, cudaMemcpyHostToDevice, st));
    // update
    rc = launch_update(ctx, S, m, sc, dt, c, chat, st, ctx->slab_scratch[j]);
    if (rc != MGRHD_OK) return rc;
    // device -> host (rho and kappa_scale are read only)
    for (int i = 0; i < 3; ++i) CU(cudaMemcpyAsync(s->mom[i] + lo, S.mom[i], w, cudaMemcpyDeviceToHost, st));
    CU(cudaMemcpyAsync(s->Egas + lo, S.Egas, w, cudaMemcpyDeviceToHost, st));
    CU(cudaMemcpy2DAsync(s->Erad + lo, pitch_h, S.Erad, pitch_d, w, Nq, cudaMemcpyDeviceToHost, st));
    for (int i = 0; i < 3; ++i)
      CU(cudaMemcpy2DAsync(s->Frad[i] + lo, pitch_h, S.Frad[i], pitch_d, w, Nq, cudaMemcpyDeviceToHost, st));
  }
  for (int k = 0; k < kSlabs; ++k) CU(cudaStreamSynchronize(ctx->slab_stream[k]));
  return MGRHD_OK;
}

static int launch_transport(mgrhd_ctx* ctx, const StatePtrs& src, const StatePtrs& dst, long long nx, double dx,
                            double wdt, double c, double chat, int bc, cudaStream_t st) {
  // two cells per thread (16-byte accesses) when every group row starts on a 16-byte boundary
  const bool v2 = nx % 2 == 0 && nx >= 4 && ((uintptr_t)src.Erad % 16 == 0) && ((uintptr_t)dst.Erad % 16 == 0) &&
                  ((uintptr_t)src.Frad[0] % 16 == 0) && ((uintptr_t)src.Frad[1] % 16 == 0) && ((uintptr_t)src.Frad[2] % 16 == 0) &&
                  ((uintptr_t)dst.Frad[0] % 16 == 0) && ((uintptr_t)dst.Frad[1] % 16 == 0) && ((uintptr_t)dst.Frad[2] % 16 == 0);
  const long long per = (v2 ? 2 : 1) * (kTransportTile - 2);
  const long long tiles = (nx + per - 1) / per;
  dim3 grid((unsigned)tiles, (unsigned)ctx->P.Nq);
  if (v2) transport_add_kernel<2><<<grid, kTransportTile, 0, st>>>(src, dst, ctx->P.closure, nx, nx, nx, wdt / dx, c, chat, bc);
  else transport_add_kernel<1><<<grid, kTransportTile, 0, st>>>(src, dst, ctx->P.closure, nx, nx, nx, wdt / dx, c, chat, bc);
  ctx->launches++;
  ctx->last_stream = st;
  CU(cudaGetLastError());
  return MGRHD_OK;
}

static int check_transport(const mgrhd_ctx* ctx, const mgrhd_state* a, const mgrhd_state* b, long long nx, double dx,
                           double c, double chat, int bc) {
  int rc = check_call(ctx, a, nx, 1.0, c, chat);
  if (rc != MGRHD_OK) return rc;
  if (!b || bc < 0 || bc > 1) return MGRHD_ERR_ARG;
  if (!(dx > 0.0)) return MGRHD_ERR_RANGE;
  if (nx > 0 && (!b->Erad || !b->Frad[0] || !b->Frad[1] || !b->Frad[2])) return MGRHD_ERR_ARG;
  if (nx > 0 && (a->Erad == b->Erad || a->Frad[0] == b->Frad[0])) return MGRHD_ERR_ARG;      // no aliasing
  if (nx > 0 && nx > (1ll << 31) * (kTransportTile - 2)) return MGRHD_ERR_ARG;
  return MGRHD_OK;
}

int mgrhd_transport_add(mgrhd_ctx* ctx, const mgrhd_state* src, const mgrhd_state* dst, long long nx, double dx,
                        double w_dt, double c, double chat, int bc, void* stream) {
  int rc = check_transport(ctx, src, dst, nx, dx, c, chat, bc);
  if (rc != MGRHD_OK) return rc;
  if (!std::isfinite(w_dt)) return MGRHD_ERR_RANGE;
  if (nx == 0) return MGRHD_OK;
  return launch_transport(ctx, to_ptrs(src), to_ptrs(dst), nx, dx, w_dt, c, chat, bc, (cudaStream_t)stream);
}

int mgrhd_imex_step_1d(mgrhd_ctx* ctx, const mgrhd_state* U, const mgrhd_state* W, long long nx, double dx, double dt,
                       double c, double chat, int bc, void* stream) {
  int rc = check_transport(ctx, U, W, nx, dx, c, chat, bc);
  if (rc != MGRHD_OK) return rc;
  if (!(dt > 0.0)) return MGRHD_ERR_RANGE;
  if (U->Srad) return MGRHD_ERR_ARG;                      // a per-update source has no place in the two stages
  if (nx > 0 && (!W->mom[0] || !W->mom[1] || !W->mom[2] || !W->Egas)) return MGRHD_ERR_ARG;
  if (nx == 0) return MGRHD_OK;
  cudaStream_t st = (cudaStream_t)stream;
  const int Nq = ctx->P.Nq;
  const size_t b1 = (size_t)nx * sizeof(double), bq = b1 * Nq;
  StatePtrs SU = to_ptrs(U), SW = to_ptrs(W);
  SW.rho = SU.rho;                                        // the work state borrows the read-only fields
  SW.kappa_scale = SU.kappa_scale;
  SW.Srad = nullptr;
  // stage 1 (Eq. 35): W = U^n + dt T(U^n), then the implicit source update with theta = 1
  for (int i = 0; i < 3; ++i) CU(cudaMemcpyAsync(SW.mom[i], SU.mom[i], b1, cudaMemcpyDeviceToDevice, st));
  CU(cudaMemcpyAsync(SW.Egas, SU.Egas, b1, cudaMemcpyDeviceToDevice, st));
  CU(cudaMemcpyAsync(SW.Erad, SU.Erad, bq, cudaMemcpyDeviceToDevice, st));
  for (int i = 0; i < 3; ++i) CU(cudaMemcpyAsync(SW.Frad[i], SU.Frad[i], bq, cudaMemcpyDeviceToDevice, st));
  rc = launch_transport(ctx, SU, SW, nx, dx, dt, c, chat, bc, st);
  if (rc != MGRHD_OK) return rc;
  rc = launch_update(ctx, SW, nx, nx, dt, c, chat, st, ctx->scratch);
  if (rc != MGRHD_OK) return rc;
  // stage 2 (Eq. 36): U = (U^n + U^(n+1/2))/2 + (dt/2) T(U^(n+1/2)), then the source update with theta = 1/2
  // (dt S(U^(n+1/2)) = U^(n+1/2) - U* and dt T(U^n) = U* - U^n turn Eq. 36's explicit part into this form)
  const int ab = ctx->sm_count * 8;
  for (int i = 0; i < 3; ++i) average_kernel<<<ab, 256, 0, st>>>(SU.mom[i], SW.mom[i], nx);
  average_kernel<<<ab, 256, 0, st>>>(SU.Egas, SW.Egas, nx);
  average_kernel<<<ab, 256, 0, st>>>(SU.Erad, SW.Erad, nx * Nq);
  for (int i = 0; i < 3; ++i) average_kernel<<<ab, 256, 0, st>>>(SU.Frad[i], SW.Frad[i], nx * Nq);
  ctx->launches += 8;
  CU(cudaGetLastError());
  rc = launch_transport(ctx, SW, SU, nx, dx, 0.5 * dt, c, chat, bc, st);
  if (rc != MGRHD_OK) return rc;
  return launch_update(ctx, SU, nx, nx, 0.5 * dt, c, chat, st, ctx->scratch);
}

int mgrhd_get_stats(mgrhd_ctx* ctx, mgrhd_stats* out) {
  if (!ctx || !out) return MGRHD_ERR_ARG;
  if (ctx->slab[0]) for (int k = 0; k < kSlabs; ++k) CU(cudaStreamSynchronize(ctx->slab_stream[k]));
  CU(cudaStreamSynchronize(ctx->last_stream));
  unsigned long long h[kStatCount];
  CU(cudaMemcpy(h, ctx->d_stats, sizeof h, cudaMemcpyDeviceToHost));
  out->n_cells = (long long)h[kStatCells];
  out->n_newton_unconverged = (long long)h[kStatNewtonUnconv];
  out->n_outer_unconverged = (long long)h[kStatOuterUnconv];
  out->n_T_nonpositive_steps = (long long)h[kStatTNonPos];
  out->n_chiF_guard = (long long)h[kStatChiFGuard];
  out->n_denominator_nonpositive = (long long)h[kStatDenNonPos];
  out->newton_evals_total = (long long)h[kStatNewtonEvals];
  out->outer_trips_total = (long long)h[kStatOuterTrips];
  out->flops = (long long)h[kStatFlops];
  for (int b = 0; b < MGRHD_HIST; ++b) {
    out->newton_hist[b] = (long long)h[kStatNewtonHist + b];
    out->outer_hist[b] = (long long)h[kStatOuterHist + b];
  }
  return MGRHD_OK;
}

int mgrhd_reset_stats(mgrhd_ctx* ctx) {
  if (!ctx) return MGRHD_ERR_ARG;
  CU(cudaMemsetAsync(ctx->d_stats, 0, kStatCount * sizeof(unsigned long long), ctx->last_stream));
  return MGRHD_OK;
}

int mgrhd_set_flop_counting(mgrhd_ctx* ctx, int on) {
  if (!ctx) return MGRHD_ERR_ARG;
  ctx->count_flops = on ? 1 : 0;
  return MGRHD_OK;
}

long long mgrhd_launch_count(const mgrhd_ctx* ctx) { return ctx ? ctx->launches : 0; }

int mgrhd_planck_edge_functions(const double* x_dev, long long n, double* yz_dev, double* xi_dev,
                                int* is_y_dev, int form, void* stream) {
  if (n < 0 || (n > 0 && (!x_dev || !yz_dev || !xi_dev || !is_y_dev)) || (form != 0 && form != 1)) return MGRHD_ERR_ARG;
  if (n == 0) return MGRHD_OK;
  CU(upload_tables_for_current_device());
  long long blocks = (n + 255) / 256;
  if (blocks > 4096) blocks = 4096;
  planck_edge_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(x_dev, n, yz_dev, xi_dev, is_y_dev, form, 0);
  CU(cudaGetLastError());
  return MGRHD_OK;
}

int mgrhd_measure_dfma_peak(long long iters, double* fma_per_second) {
  if (!fma_per_second || iters < 8) return MGRHD_ERR_ARG;
  int dev = 0, sms = 0;
  CU(cudaGetDevice(&dev));
  CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  double* d_out = nullptr;
  CU(cudaMalloc(&d_out, sizeof(double)));
  cudaEvent_t e0, e1;
  CU(cudaEventCreate(&e0));
  CU(cudaEventCreate(&e1));
  const int blocks = sms * 8, threads = 256;
  iters = (iters / 8) * 8;
  dfma_peak_kernel<<<blocks, threads>>>(iters / 16, d_out);   // warm-up
  float best = 1e30f;
  for (int r = 0; r < 3; ++r) {
    CU(cudaEventRecord(e0));
    dfma_peak_kernel<<<blocks, threads>>>(iters, d_out);
    CU(cudaEventRecord(e1));
    CU(cudaEventSynchronize(e1));
    float ms = 0.f;
    CU(cudaEventElapsedTime(&ms, e0, e1));
    if (ms < best) best = ms;
  }
  CU(cudaGetLastError());
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(d_out);
  *fma_per_second = (double)blocks * threads * (double)iters / (best * 1e-3);
  return MGRHD_OK;
}

// ---- mgrhd_source_update_static: the update without any device allocation (include/mgrhd.h) ---------------------
// The scratch and the counter block of the update kernel as file-scope device arrays.  In HOST code these names are
// host-side stand-ins, not device addresses: the addresses the kernel gets come from cudaGetSymbolAddress, once per
// device, with that device current (static_setup below).
static __device__ __align__(256) double g_static_scratch[MGRHD_STATIC_SCRATCH_BYTES / sizeof(double)];
static __device__ __align__(256) unsigned long long g_static_stats[kStatCount];

struct StaticDev {
  std::once_flag once;
  cudaError_t err;
  double* scratch;
  unsigned long long* stats;
  int sm_count;
};
static StaticDev g_static_dev[16];

static cudaError_t static_setup(int dev) {
  StaticDev& d = g_static_dev[dev];
  std::call_once(d.once, [&d, dev]() {
    d.err = upload_tables_for_current_device();
    if (d.err == cudaSuccess) d.err = cudaDeviceGetAttribute(&d.sm_count, cudaDevAttrMultiProcessorCount, dev);
    if (d.err == cudaSuccess) d.err = cudaGetSymbolAddress((void**)&d.scratch, g_static_scratch);
    if (d.err == cudaSuccess) d.err = cudaGetSymbolAddress((void**)&d.stats, g_static_stats);
  });
  return d.err;
}

int mgrhd_source_update_static(const double* edges, int Nq, const mgrhd_units* u, const mgrhd_opacity_model* m,
                               const mgrhd_state* s, long long n, double dt, double c, double chat, void* stream,
                               mgrhd_stats* stats_out) {
  // the checks of mgrhd_init for the models the tuned kernel runs
  if (!edges || !u || !m) return MGRHD_ERR_ARG;
  if (m->spectrum != 0 || m->outer_mode != 0 || (m->opacity_kind != 0 && m->opacity_kind != 1)) return MGRHD_ERR_ARG;
  if (!m->kappa_lo || !m->alpha || Nq < 1 || Nq > MGRHD_MAX_GROUPS) return MGRHD_ERR_ARG;
  if (m->closure < 0 || m->closure > 1 || m->outer_stop < 0 || m->outer_stop > 1 || m->newton_maxit < 1 ||
      m->outer_maxit < 1)
    return MGRHD_ERR_ARG;
  if (!(u->a_rad > 0) || !(u->k_B > 0) || !(u->h_planck > 0) || !(u->mean_mass > 0) || !(u->gamma > 1) ||
      !(m->newton_tol > 0) || !(m->outer_tol > 0))
    return MGRHD_ERR_RANGE;
  if (m->opacity_kind == 1 && (!(m->T_ref > 0) || !std::isfinite(m->T_ref) || !std::isfinite(m->p_T))) return MGRHD_ERR_RANGE;
  for (int g = 0; g < Nq; ++g) {
    if (!(edges[g] >= 0.0) || !(edges[g + 1] > edges[g])) return MGRHD_ERR_EDGES;
    if (m->alpha[g] != 0.0 && (edges[g] == 0.0 || std::isinf(edges[g + 1]))) return MGRHD_ERR_ALPHA;
    if (!std::isfinite(m->alpha[g]) || !(m->kappa_lo[g] > 0.0) || !std::isfinite(m->kappa_lo[g])) return MGRHD_ERR_RANGE;
  }
  // a context on the host stack: parameter block as mgrhd_init fills it, nothing on the device
  mgrhd_ctx ctx;
  std::memset(&ctx, 0, sizeof ctx);
  Params& P = ctx.P;
  P.Nq = Nq;
  P.closure = m->closure;
  P.newton_maxit = m->newton_maxit;
  P.outer_maxit = m->outer_maxit;
  P.outer_stop = m->outer_stop;
  P.newton_tol = m->newton_tol;
  P.outer_tol = m->outer_tol;
  P.outer_rel_tol = m->outer_rel_tol;
  P.a_rad = u->a_rad;
  P.h_over_k = u->h_planck / u->k_B;
  P.cv_over_rho = u->k_B / ((u->gamma - 1.0) * u->mean_mass);
  for (int g = 0; g <= Nq; ++g) P.nu[g] = edges[g];
  P.inv_T_ref = m->opacity_kind == 1 ? 1.0 / m->T_ref : 1.0;
  P.p_T = m->opacity_kind == 1 ? m->p_T : 0.0;
  ctx.G.opacity_kind = m->opacity_kind;
  for (int g = 0; g < Nq; ++g) {
    const double a = m->alpha[g], k = m->kappa_lo[g];
    P.alpha[g] = a;
    P.k_lo[g] = k;
    if (a == 0.0) {                       // piecewise constant, Eq. 17
      P.k_hi[g] = k;
      P.k_mean[g] = k;
    } else {                              // Eq. 19 at nu_g+; Eq. 30 with alpha_Q = -1
      const double z = a * std::log(edges[g + 1] / edges[g]);
      P.k_hi[g] = k * std::exp(z);
      P.k_mean[g] = k * (std::expm1(z) / z);
    }
    P.inv_k_mean[g] = 1.0 / P.k_mean[g];
    P.k_num[g] = P.k_mean[g] * ((4.0 + a) / 3.0);
    P.onepa[g] = 1.0 + a;
  }
  CU(cudaGetDevice(&ctx.device));
  if (ctx.device < 0 || ctx.device >= 16) return MGRHD_ERR_ARG;
  int rc = check_call(&ctx, s, n, dt, c, chat);
  if (rc != MGRHD_OK) return rc;
  CU(static_setup(ctx.device));
  const StaticDev& d = g_static_dev[ctx.device];
  ctx.sm_count = d.sm_count;
  ctx.d_stats = d.stats;
  CU(configure_ctx(&ctx));             // function attributes and occupancy of the instantiation: no allocation
  // the grid launch_update will use, and the scratch it indexes: head + 3 NQL doubles per thread of the grid
  long long blocks = (long long)ctx.sm_count * ctx.cfg_bps;
  const long long cells_per_cta = ctx.cfg_threads / ctx.cfg_l;
  const long long want = (n + cells_per_cta - 1) / cells_per_cta;
  if (blocks > want) blocks = want;
  const long long need = (long long)(kScratchHead * sizeof(double)) + 3ll * ctx.cfg_nq * (long long)sizeof(double) * blocks * ctx.cfg_threads;
  if (need > MGRHD_STATIC_SCRATCH_BYTES) {
    std::snprintf(g_err, sizeof g_err,
                  "mgrhd_source_update_static: Nq = %d, ncells = %lld needs %lld bytes of scratch, the static array holds %lld; "
                  "use mgrhd_source_update or fewer cells per call",
                  Nq, n, need, (long long)MGRHD_STATIC_SCRATCH_BYTES);
    return MGRHD_ERR_SIZE;
  }
  const cudaStream_t st = (cudaStream_t)stream;
  CU(cudaMemsetAsync(d.stats, 0, kStatCount * sizeof(unsigned long long), st));   // counters of this call only
  if (n > 0) {
    rc = launch_update(&ctx, to_ptrs(s), n, n, dt, c, chat, st, d.scratch);      // (clears the work counter itself)
    if (rc != MGRHD_OK) return rc;
  }
  if (stats_out) {
    ctx.last_stream = st;
    return mgrhd_get_stats(&ctx, stats_out);
  }
  return MGRHD_OK;
}

void mgrhd_free(mgrhd_ctx* ctx) {
  if (!ctx) return;
  for (int k = 0; k < kSlabs; ++k) {
    if (ctx->slab[k]) cudaFree(ctx->slab[k]);
    if (ctx->slab_scratch[k]) cudaFree(ctx->slab_scratch[k]);
    if (ctx->slab_stream[k]) cudaStreamDestroy(ctx->slab_stream[k]);
  }
  if (ctx->d_stats) cudaFree(ctx->d_stats);
  if (ctx->scratch) cudaFree(ctx->scratch);
  if (ctx->d_lnk) cudaFree(ctx->d_lnk);
  delete ctx;
}

}  // extern "C"
