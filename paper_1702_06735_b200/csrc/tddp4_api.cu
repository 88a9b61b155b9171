// tddp4_api.cu -- the C-ABI of include/tddp4.h: handle, host-side model analysis, dirty tracking,
// launch sequencing.  Every arithmetic step of the hot path runs in the kernels of kernels.cuh; the host
// only derives per-call scalars (pole constants of the lineshapes, time integrals) in fp64.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <cstdlib>
#include <limits>
#include <string>
#include <type_traits>
#include <vector>

#include "../../include/tddp4.h"
#include "kernels.cuh"
#include "grad_kernels.cuh"

using namespace tddp4k;

namespace {

constexpr int N_SLOTS = 64;
constexpr int SLOT_DOUBLES = 8;

struct EventSet {
  int64_t n = 0, ld = 0;
  double *cache = nullptr;                           // static cache, tile-major (tables.h): s, g, f [, w] rows
  int R = 0;                                         // rows per tile
  double2 *a = nullptr;                              // coupling columns [K_c][ld]
  double *t = nullptr, *sigma_t = nullptr, *w = nullptr;
  double *tr = nullptr;                              // resolution mode: time rows psi[4], tint[4], [8][ld]
  bool tres_valid = false;                           // tr matches the current x, y, tau
  int tres_parts = 3;                                // which halves of tr are stale: bit 0 real-lambda rows (y, tau), bit 1 complex (x, tau)
  double *trg = nullptr;                             // derivative rows of the gradient in resolution mode, [8][ld] (on demand)
  bool tresg_valid = false;
  double sum_t = 0.0, t_max = 0.0;                   // sum and max |t| of the decay times (fixed-order kernel)
  double sig_lo = 0.0, sig_hi = 0.0;                 // range of sigma_t (resolution mode: the window-integral table covers it)
  bool cols_dirty = true;                            // coupling columns stale (a mass or width moved since they were built)
  bool loaded = false;
};

struct ProfEvent { int id; cudaEvent_t a, b; double bytes; };

}  // namespace

struct tddp4 {
  int device = 0;
  cudaStream_t stream = nullptr;
  bool own_stream = false;
  ModelTab M{};
  StreamTab S{};                     // the same model, flattened for the per-call kernels
  uint32_t store_mask = 0xFFFFFFFFu; // coupling columns of the data sample whose stored values are stale (bit = column)
  int prev_kind = 0;                 // last per-call kernel enqueued with nothing after it: 0 none/other, 1 NLL, 2 COLNLL, 3 GRAM
  int size_class = 0;                // load-batch sizes (GI, GT) of the per-call kernels: 0 (4,4), 1 (8,8), 2 (12,16)
  std::vector<tddp4_res> res;
  std::vector<tddp4_term> terms;   // caller's order
  double t_lo = 0.0, t_hi = INFINITY;
  int use_resolution = 0;
  // parameters
  bool have_params = false;
  LineParams LP{};
  RateParams RP{};
  FaddTab FT{};                      // Faddeeva expansion coefficients (resolution mode)
  double *staging = nullptr;         // device staging of host four-momenta (grow-only)
  size_t staging_cap = 0;
  TresTable *tres_tab = nullptr;     // device: Chebyshev table of the window integrals in sigma, rebuilt with the time rows
  std::vector<double> mass, width;
  EventSet set[2];
  // normalisation
  double *G = nullptr;               // device [K_c][K_c][2] sums
  bool gram_valid = false;           // G matches the current masses/widths
  bool gram_overridden = false;
  int64_t gram_n = 0;                // event count G is normalised by
  // scratch
  double *partials = nullptr;
  size_t partials_cap = 0;
  unsigned int *ticket = nullptr;
  double *results = nullptr;         // device [N_SLOTS][SLOT_DOUBLES]
  double *results_host = nullptr;    // pinned host slots; the NLL kernels write them directly (zero-copy) ...
  double *results_host_dev = nullptr; // ... through this device alias
  cudaEvent_t slot_event[N_SLOTS] = {nullptr};
  bool slot_used[N_SLOTS] = {false};
  double *grad_host = nullptr, *grad_host_dev = nullptr;   // mapped pinned result of tddp4_nll_grad: [GRAD_OFFSET + 4 K_c + 2]
  double *batch_res = nullptr;       // device [batch_cap][SLOT_DOUBLES]
  double *batch_res_host = nullptr;  // pinned mirror
  int64_t batch_cap = 0;
  // generator scratch
  uint32_t *gen_flags = nullptr, *gen_counts = nullptr;
  unsigned long long *gen_offs = nullptr, *gen_scalars = nullptr;   // [0] pilot max bits, [1] overflow
  int64_t gen_cap = 0;
  // profiling
  bool profiling = false;
  std::vector<ProfEvent> pending;
  std::vector<cudaEvent_t> pool;
  double prof_ms[TDDP4_K_COUNT] = {0};
  double prof_bytes[TDDP4_K_COUNT] = {0};   // algorithmic bytes of the profiled launches
  int64_t prof_n[TDDP4_K_COUNT] = {0};
  int64_t launches = 0;
  double seq = 0.0;                  // sequence stamp of the last NLL kernel enqueued (word [5] of its result slot)
  bool stamp = false;                // the evaluation being enqueued writes to a polled slot: its kernel carries a stamp
  double slot_seq[N_SLOTS] = {0};    // stamp each slot is waiting for
  int sm_count = 148;
  std::string err;
};

namespace {

int fail(tddp4 *h, int code, const char *fmt, ...) {
  if (h) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    h->err = buf;
  }
  return code;
}

#define CU(call)                                                                                   \
  do {                                                                                             \
    cudaError_t e_ = (call);                                                                       \
    if (e_ != cudaSuccess) return fail(h, TDDP4_ERR_CUDA, "%s: %s", #call, cudaGetErrorString(e_)); \
  } while (0)

struct Prof {   // RAII: CUDA events around one launch when profiling is on
  tddp4 *h; int id; double bytes; cudaEvent_t a = nullptr, b = nullptr;
  Prof(tddp4 *h_, int id_, double bytes_ = 0.0) : h(h_), id(id_), bytes(bytes_) {
    ++h->launches;
    if (!h->profiling) return;
    auto get = [&]() { cudaEvent_t e; if (!h->pool.empty()) { e = h->pool.back(); h->pool.pop_back(); } else cudaEventCreate(&e); return e; };
    a = get(); b = get();
    cudaEventRecord(a, h->stream);
  }
  ~Prof() {
    if (!a) return;
    cudaEventRecord(b, h->stream);
    h->pending.push_back({id, a, b, bytes});
  }
};

void drain_profile(tddp4 *h) {
  for (auto &p : h->pending) {
    cudaEventSynchronize(p.b);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, p.a, p.b);
    h->prof_ms[p.id] += ms;
    h->prof_n[p.id] += 1;
    h->prof_bytes[p.id] += p.bytes;
    h->pool.push_back(p.a);
    h->pool.push_back(p.b);
  }
  h->pending.clear();
}

int parent_L(int sf) {
  switch (sf) {
    case SF_VV_S: return 0; case SF_VV_P: return 1; case SF_VV_D: return 2;
    case SF_AP_S: return 1; case SF_TP_D: return 2; case SF_AP_D: return 1; default: return 0;
  }
}

int find_or_add_sys(ModelTab &M, unsigned mask) {
  for (int i = 0; i < M.n_sys; ++i)
    if (M.sys_mask[i] == mask) return i;
  if (M.n_sys >= MAX_SYS) return -1;
  M.sys_mask[M.n_sys] = (uint8_t)mask;
  return M.n_sys++;
}

int find_or_add_inst(ModelTab &M, const InstTab &in) {
  for (int i = 0; i < M.n_inst; ++i) {
    const InstTab &o = M.inst[i];
    if (o.res == in.res && o.sys == in.sys && o.sub == in.sub && o.dres == in.dres && o.ma == in.ma && o.mb == in.mb && o.L == in.L)
      return i;
  }
  if (M.n_inst >= MAX_INST) return -1;
  M.inst[M.n_inst] = in;
  return M.n_inst++;
}

double host_breakup(double M, double ma, double mb) {
  double rad = (M - ma - mb) * (M + ma + mb) * (M + ma - mb) * (M - ma + mb);
  return rad > 0.0 ? std::sqrt(rad) / (2.0 * M) : 0.0;
}
double host_barrier2(int L, double z) {   // F_L(z)^2
  if (L == 0) return 1.0;
  if (L == 1) return 1.0 / (1.0 + z);
  return 1.0 / (9.0 + 3.0 * z + z * z);
}

// O-8: window integrals of e^{-Gamma t}{cosh, cos, sinh, sin}
void time_integrals(double x, double y, double Gamma, double lo, double hi, double T[4]) {
  using cd = std::complex<double>;
  auto I = [&](cd lam) {
    cd a = std::exp(-lam * lo);
    cd b = std::isinf(hi) ? cd(0.0, 0.0) : std::exp(-lam * hi);
    return (a - b) / lam;
  };
  cd Im = I(cd(Gamma * (1.0 - y), 0.0)), Ip = I(cd(Gamma * (1.0 + y), 0.0)), Ix = I(cd(Gamma, -Gamma * x));
  T[0] = 0.5 * (Im.real() + Ip.real());
  T[1] = Ix.real();
  T[2] = 0.5 * (Im.real() - Ip.real());
  T[3] = Ix.imag();
}

// d/dx and d/dy of those integrals: dI/dlambda = (-lo e^{-lambda lo} + hi e^{-lambda hi}) / lambda - I / lambda,
// d lambda-+ / dy = -+Gamma, d lambda_x / dx = -i Gamma
GradParams time_integral_derivatives(double x, double y, double Gamma, double lo, double hi) {
  using cd = std::complex<double>;
  auto dI = [&](cd lam) {
    cd a = std::exp(-lam * lo);
    cd b = std::isinf(hi) ? cd(0.0, 0.0) : std::exp(-lam * hi);
    cd hb = std::isinf(hi) ? cd(0.0, 0.0) : hi * b;
    cd I = (a - b) / lam;
    return (-lo * a + hb) / lam - I / lam;
  };
  cd dm = dI(cd(Gamma * (1.0 - y), 0.0)), dp = dI(cd(Gamma * (1.0 + y), 0.0)), dx = dI(cd(Gamma, -Gamma * x));
  cd ddx = cd(0.0, -Gamma) * dx;
  GradParams g;
  g.dT1dx = ddx.real();
  g.dT3dx = ddx.imag();
  g.dT0dy = 0.5 * (-Gamma * dm.real() + Gamma * dp.real());
  g.dT2dy = 0.5 * (-Gamma * dm.real() - Gamma * dp.real());
  return g;
}

int ensure_partials(tddp4 *h, size_t doubles) {
  if (doubles <= h->partials_cap) return TDDP4_OK;
  if (h->partials) cudaFree(h->partials);
  h->partials = nullptr;
  h->partials_cap = 0;
  CU(cudaMalloc(&h->partials, doubles * sizeof(double)));
  h->partials_cap = doubles;
  return TDDP4_OK;
}

void free_set(EventSet &e) {
  cudaFree(e.cache); cudaFree(e.a); cudaFree(e.t); cudaFree(e.sigma_t); cudaFree(e.w); cudaFree(e.tr); cudaFree(e.trg);
  e = EventSet{};
}

int stream_grid(const tddp4 *h, int64_t n) {
  return (int)std::max<int64_t>(1, std::min<int64_t>((n + STREAM_BLOCK - 1) / STREAM_BLOCK,
                                                     (int64_t)h->sm_count * STREAM_BLOCKS_PER_SM));
}

// algorithmic bytes per event of the step-1 caches a dirty call has to read: s rows in use, g rows, f rows
double static_bytes_per_event(const tddp4 *h) { return 8.0 * (h->M.n_su + h->M.n_inst + h->M.n_terms); }

// size classes of the per-call kernels (stream_kernels.cuh): f(GI, GT) with compile-time constants
template <class F>
auto with_size_class(int cls, F &&f) {
  switch (cls) {
    case 0: return f(std::integral_constant<int, 4>{}, std::integral_constant<int, 4>{});
    case 1: return f(std::integral_constant<int, 8>{}, std::integral_constant<int, 8>{});
    default: return f(std::integral_constant<int, 12>{}, std::integral_constant<int, 16>{});
  }
}

// launch with programmatic stream serialization (stream_kernels.cuh, pdl_*): the kernel may become resident while its
// predecessor in the stream drains; it synchronises with it through griddepcontrol.wait
template <class... KArgs, class... Args>
cudaError_t launch_pdl(void (*kernel)(KArgs...), int grid, int block, size_t smem, cudaStream_t stream, Args &&...args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)grid);
  cfg.blockDim = dim3((unsigned)block);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
}
// a failed launch leaves the handle's bookkeeping untouched (nothing was enqueued): the caller may retry
#define CU_LAUNCH(expr)                                                                              \
  do {                                                                                               \
    cudaError_t e_ = (expr);                                                                         \
    if (e_ != cudaSuccess) return fail(h, TDDP4_ERR_CUDA, "kernel launch: %s", cudaGetErrorString(e_)); \
  } while (0)
enum { PREV_NONE = 0, PREV_NLL = 1, PREV_COLNLL = 2, PREV_GRAM = 3 };

template <int NB>
int launch_gram(tddp4 *h, const EventSet &e) {
  const ModelTab &M = h->M;
  int grid = stream_grid(h, e.n);
  int rc = ensure_partials(h, (size_t)(grid + (grid + GRAM_GROUP - 1) / GRAM_GROUP) * 64 * NB * NB + 16);
  if (rc) return rc;
  StreamTab S = h->S;
  S.R = e.R;
  S.w_off = e.w ? (M.n_sys + S.n_inst4 + S.n_terms4) * 32 : -1;
  Prof p(h, TDDP4_K_GRAM, (double)e.n * (static_bytes_per_event(h) + (e.w ? 8.0 : 0.0)));
  CU_LAUNCH(with_size_class(h->size_class, [&](auto ni, auto nt) {
    return launch_pdl(gram_stream_kernel<NB, decltype(ni)::value, decltype(nt)::value>, grid, STREAM_BLOCK,
                      gram_smem_bytes(NB, S.n_inst4), h->stream, S, h->LP, (const double *)e.cache, e.n, h->partials, h->ticket, h->G);
  }));
  h->prev_kind = PREV_GRAM;
  return TDDP4_OK;
}

// step 6: refresh the Gram matrix of this handle's normalisation sample if masses/widths changed
int ensure_gram(tddp4 *h) {
  if (h->gram_valid) return TDDP4_OK;
  EventSet &e = h->set[1];
  if (!e.loaded) return fail(h, TDDP4_ERR_STATE, "normalisation sample not loaded");
  int KC = h->M.n_kc, rc;
  if (KC <= 4) rc = launch_gram<1>(h, e);
  else if (KC <= 8) rc = launch_gram<2>(h, e);
  else if (KC <= 12) rc = launch_gram<3>(h, e);
  else rc = launch_gram<4>(h, e);
  if (rc) return rc;
  CU(cudaGetLastError());
  h->gram_valid = true;
  h->gram_overridden = false;
  h->gram_n = e.n;
  return TDDP4_OK;
}

template <int KC>
int launch_nll(tddp4 *h, const EventSet &e, double inv_n, double *result, bool small) {
  int grid = stream_grid(h, e.n);
  int rc = ensure_partials(h, (size_t)3 * grid + 16);
  if (rc) return rc;
  Prof p(h, TDDP4_K_NLL, (double)e.n * (16.0 * KC + 8.0));
  // the columns and t are untouched by a preceding NLL or Gram kernel: only the final reduction has to wait for it
  const int early = !(h->prev_kind == PREV_NLL || h->prev_kind == PREV_GRAM);
  if (small)
    CU_LAUNCH(launch_pdl(nll_stream_kernel<KC, true>, grid, STREAM_BLOCK, 0, h->stream, (const double2 *)e.a, (const double *)e.t, e.ld, e.n, h->RP,
                         (const double *)h->G, inv_n, e.sum_t, h->partials, h->ticket, result, early, h->stamp ? ++h->seq : 0.0));
  else
    CU_LAUNCH(launch_pdl(nll_stream_kernel<KC, false>, grid, STREAM_BLOCK, 0, h->stream, (const double2 *)e.a, (const double *)e.t, e.ld, e.n, h->RP,
                         (const double *)h->G, inv_n, e.sum_t, h->partials, h->ticket, result, early, h->stamp ? ++h->seq : 0.0));
  h->prev_kind = PREV_NLL;
  return TDDP4_OK;
}

template <int KC>
int launch_nll_res(tddp4 *h, const EventSet &e, double inv_n, double *result) {
  int grid = stream_grid(h, e.n);
  int rc = ensure_partials(h, (size_t)3 * grid + 16);
  if (rc) return rc;
  Prof p(h, TDDP4_K_NLL, (double)e.n * (16.0 * KC + 64.0));
  CU_LAUNCH(launch_pdl(nll_res_kernel<KC>, grid, STREAM_BLOCK, 0, h->stream, (const double2 *)e.a, (const double *)e.tr, e.ld, e.n, h->RP,
                       (const double *)h->G, inv_n, h->partials, h->ticket, result, h->stamp ? ++h->seq : 0.0));
  h->prev_kind = PREV_NLL;
  return TDDP4_OK;
}

int launch_colnll(tddp4 *h, const EventSet &e, double inv_n, double *result, bool small) {
  const ModelTab &M = h->M;
  int grid = stream_grid(h, e.n);
  int rc = ensure_partials(h, (size_t)3 * grid + 16);
  if (rc) return rc;
  StreamTab S = h->S;
  S.R = e.R;
  size_t smem = colnll_smem_bytes(S.n_inst4);
  int n_stored = 0;                      // columns actually rewritten by this launch
  for (int kap = 0; kap < M.n_kc; ++kap) n_stored += (h->store_mask >> kap) & 1u;
  Prof p(h, TDDP4_K_COLNLL, (double)e.n * (static_bytes_per_event(h) + (h->use_resolution ? 64.0 : 8.0) + 16.0 * n_stored));
  const int mode = h->use_resolution ? 2 : (small ? 1 : 0);
  const int early = h->prev_kind != PREV_GRAM;   // a Gram kernel neither reads nor writes the columns this kernel rewrites
  const double sum_t = h->use_resolution ? 0.0 : e.sum_t;
  const double *tp = h->use_resolution ? e.tr : e.t;
#define COLNLL_LAUNCH(SM, RS)                                                                                                  \
  launch_pdl(colnll_stream_kernel<SM, RS, NI, NT>, grid, STREAM_BLOCK, smem, h->stream, S, h->LP, (const double *)e.cache, tp, e.ld, e.n, \
             e.a, h->RP, (const double *)h->G, inv_n, sum_t, h->partials, h->ticket, result, early, h->store_mask, seq)
  const double seq = h->stamp ? h->seq + 1.0 : 0.0;
  cudaError_t launched = with_size_class(h->size_class, [&](auto ni, auto nt) {
    constexpr int NI = decltype(ni)::value, NT = decltype(nt)::value;
    if (mode == 2) return COLNLL_LAUNCH(false, true);
    if (mode == 1) return COLNLL_LAUNCH(true, false);
    return COLNLL_LAUNCH(false, false);
  });
#undef COLNLL_LAUNCH
  CU_LAUNCH(launched);
  if (h->stamp) h->seq = seq;
  h->prev_kind = PREV_COLNLL;   // committed only after the launch succeeded: a failed launch keeps the stale-column set
  h->store_mask = 0;
  return TDDP4_OK;
}

int dispatch_nll(tddp4 *h, EventSet &d, bool fused, double inv_n, double *result, bool small) {
  int rc;
  if (fused) {
    rc = launch_colnll(h, d, inv_n, result, small);
  } else {
    switch (h->M.n_kc) {
#define CASE(k) case k: rc = h->use_resolution ? launch_nll_res<k>(h, d, inv_n, result) : launch_nll<k>(h, d, inv_n, result, small); break;
      CASE(1) CASE(2) CASE(3) CASE(4) CASE(5) CASE(6) CASE(7) CASE(8) CASE(9) CASE(10) CASE(11) CASE(12)
      CASE(13) CASE(14) CASE(15) CASE(16)
#undef CASE
      default: return fail(h, TDDP4_ERR_ARG, "unsupported number of couplings %d", h->M.n_kc);
    }
  }
  if (rc) return rc;
  CU(cudaGetLastError());
  return TDDP4_OK;
}

// inspection path: coupling columns of the data set for the current masses/widths, no normalisation needed
int enqueue_columns_only(tddp4 *h) {
  EventSet &d = h->set[0];
  int rc = dispatch_nll(h, d, true, 0.0, h->results + (size_t)N_SLOTS * SLOT_DOUBLES, false);
  if (rc) return rc;
  d.cols_dirty = false;
  return TDDP4_OK;
}

// steps 2..7 for the current parameters; result: device [SLOT_DOUBLES]; prob: device [n] or NULL
int enqueue_nll(tddp4 *h, double *result, double *prob) {
  if (!h->have_params) return fail(h, TDDP4_ERR_STATE, "tddp4_set_params has not been called");
  EventSet &d = h->set[0];
  if (!d.loaded) return fail(h, TDDP4_ERR_STATE, "data sample not loaded");
  int rc = ensure_gram(h);
  if (rc) return rc;
  if (h->use_resolution && !d.tres_valid && d.n > 0) {   // x, y, tau or the sample changed: rebuild the time rows
    int grid = (int)((d.n + TRES_BLOCK - 1) / TRES_BLOCK);
    if (h->use_resolution == 2) {          // time-integrated: the rows are the window integrals, the same for every event
      Row8 v;
      for (int m = 0; m < 4; ++m) v.v[m] = v.v[4 + m] = h->RP.T[m];
      Prof p(h, TDDP4_K_TRES, (double)d.n * 64.0);
      fill_rows_kernel<<<(int)((d.n + 255) / 256), 256, 0, h->stream>>>(d.tr, d.ld, d.n, v);
    } else {
      Prof p(h, TDDP4_K_TRES, (double)d.n * 80.0);
      tres_table_kernel<<<1, 32, 0, h->stream>>>(h->FT, h->RP.x, h->RP.y, h->RP.Gamma, h->t_lo, h->t_hi, d.sig_lo, d.sig_hi, h->tres_tab);
      tres_kernel<<<grid, TRES_BLOCK, 0, h->stream>>>(h->FT, d.t, d.sigma_t, d.n, h->RP.x, h->RP.y, h->RP.Gamma, h->t_lo, h->t_hi,
                                                      h->tres_tab, d.tr, d.ld, d.tres_parts);
      ++h->launches;
    }
    CU(cudaGetLastError());
    d.tres_valid = true;
    d.tres_parts = 0;
  }
  double inv_n = h->gram_n > 0 ? 1.0 / (double)h->gram_n : 0.0;
  // Taylor forms of the four time functions are valid when both mixing phases stay below 1/4 on this sample
  const RateParams &R = h->RP;
  bool small = std::fabs(R.y) * R.Gamma * d.t_max < 0.25 && std::fabs(R.x) * R.Gamma * d.t_max < 0.25;
  if (d.cols_dirty && d.n > 0) {
    // columns stale: the fused kernel rebuilds them and finishes the NLL in the same pass
    rc = dispatch_nll(h, d, true, inv_n, result, small);
    if (rc) return rc;
    d.cols_dirty = false;
  } else {
    rc = dispatch_nll(h, d, false, inv_n, result, small);
    if (rc) return rc;
  }
  if (prob && d.n > 0) {   // per-event probabilities from the columns and the N the NLL kernel has just written
    int grid = (int)((d.n + STREAM_BLOCK - 1) / STREAM_BLOCK);
    ++h->launches;
    if (h->use_resolution)
      prob_res_kernel<<<grid, STREAM_BLOCK, 0, h->stream>>>(d.a, d.tr, d.ld, d.n, h->M.n_kc, h->RP, h->G, inv_n, prob);
    else if (small) prob_kernel<true><<<grid, STREAM_BLOCK, 0, h->stream>>>(d.a, d.t, d.ld, d.n, h->M.n_kc, h->RP, result, prob);
    else prob_kernel<false><<<grid, STREAM_BLOCK, 0, h->stream>>>(d.a, d.t, d.ld, d.n, h->M.n_kc, h->RP, result, prob);
    CU(cudaGetLastError());
  }
  return TDDP4_OK;
}

int enqueue_nll_slot(tddp4 *h, int slot, double *prob) {
  // without prob_out the last block writes its five doubles straight into the pinned host slot: no copy on the
  // critical path of a synchronous call.  With prob_out the probability kernel reads N back from the slot, so the slot
  // stays in device memory and is copied.
  const bool direct = prob == nullptr;
  double *result = (direct ? h->results_host_dev : h->results) + (size_t)slot * SLOT_DOUBLES;
  h->stamp = direct;
  int rc = enqueue_nll(h, result, prob);
  h->stamp = false;
  if (rc) return rc;
  if (!direct)
    CU(cudaMemcpyAsync(h->results_host + (size_t)slot * SLOT_DOUBLES, result, SLOT_DOUBLES * sizeof(double),
                       cudaMemcpyDeviceToHost, h->stream));
  CU(cudaEventRecord(h->slot_event[slot], h->stream));
  h->slot_used[slot] = true;
  h->slot_seq[slot] = direct ? h->seq : 0.0;
  return TDDP4_OK;
}

// Wait for a result slot.  A slot in mapped host memory carries the kernel's sequence stamp in word [5], written after
// the result behind a system-wide fence: the host polls that word (about a microsecond after the kernel's last store)
// instead of going through cudaEventSynchronize (measured: 36 -> 2x us per synchronous coupling-only call).  The event
// is still consulted from time to time so that a failed kernel cannot hang the caller.
int wait_slot(tddp4 *h, int slot) {
  const double want = h->slot_seq[slot];
  if (want > 0.0) {
    const volatile double *flag = h->results_host + (size_t)slot * SLOT_DOUBLES + 5;
    for (long spin = 0;; ++spin) {
      if (*flag == want) return TDDP4_OK;
      if ((spin & 0xfff) == 0xfff) {
        cudaError_t q = cudaEventQuery(h->slot_event[slot]);
        if (q == cudaSuccess) break;                       // complete: the stamp is visible by now (or the launch never ran)
        if (q != cudaErrorNotReady) return fail(h, TDDP4_ERR_CUDA, "cudaEventQuery: %s", cudaGetErrorString(q));
      }
    }
  }
  CU(cudaEventSynchronize(h->slot_event[slot]));
  return TDDP4_OK;
}

// gradient kernels (grad_kernels.cuh): whole warps iterate together, per-warp X and W tiles in dynamic shared memory
template <int KC>
int launch_nll_grad_res(tddp4 *h, const EventSet &e, double inv_n) {
  constexpr int NB = grad_nb<KC>();
  int grid = stream_grid(h, e.n);
  int rc = ensure_partials(h, (size_t)grid * (NB * 32 + 9) + 16);
  if (rc) return rc;
  const size_t smem = grad_smem_bytes<KC>();
  Prof p(h, TDDP4_K_GRAD, (double)e.n * (16.0 * KC + 128.0));
  nll_grad_res_kernel<KC><<<grid, STREAM_BLOCK, smem, h->stream>>>(e.a, e.tr, e.trg, e.ld, e.n, h->RP, h->G, inv_n, h->partials, h->ticket,
                                                                  h->grad_host_dev);
  return TDDP4_OK;
}

template <int KC>
int launch_nll_grad(tddp4 *h, const EventSet &e, double inv_n, bool small) {
  constexpr int NB = grad_nb<KC>();
  int grid = (int)std::max<int64_t>(1, std::min<int64_t>((e.n + STREAM_BLOCK - 1) / STREAM_BLOCK, (int64_t)h->sm_count * grad_bps<KC>()));
  int rc = ensure_partials(h, (size_t)grid * (NB * 32 + 5) + 16);
  if (rc) return rc;
  GradParams gp = time_integral_derivatives(h->RP.x, h->RP.y, h->RP.Gamma, h->t_lo, h->t_hi);
  const size_t smem = grad_smem_bytes<KC>();
  Prof p(h, TDDP4_K_GRAD, (double)e.n * (16.0 * KC + 8.0));
  if (small)
    nll_grad_kernel<KC, true><<<grid, STREAM_BLOCK, smem, h->stream>>>(e.a, e.t, e.ld, e.n, h->RP, gp, h->G, inv_n, e.sum_t, h->partials,
                                                                      h->ticket, h->grad_host_dev);
  else
    nll_grad_kernel<KC, false><<<grid, STREAM_BLOCK, smem, h->stream>>>(e.a, e.t, e.ld, e.n, h->RP, gp, h->G, inv_n, e.sum_t, h->partials,
                                                                       h->ticket, h->grad_host_dev);
  return TDDP4_OK;
}

}  // namespace

// =====================================================================================================
extern "C" {

const char *tddp4_version(void) { return "tddp4 0.1 (sm_100a, fp64)"; }

const char *tddp4_last_error(const tddp4 *h) { return h ? h->err.c_str() : "null handle"; }

int tddp4_create(const tddp4_model_desc *desc, tddp4 **out) {
  if (!desc || !out) return TDDP4_ERR_ARG;
  *out = nullptr;
  tddp4 *h = new tddp4;
  auto bail = [&](int code) { *out = h; return code; };   // handle kept so the caller can read the error text
  if (desc->n_res < 0 || desc->n_res > TDDP4_MAX_RES || desc->n_terms < 1 || desc->n_terms > TDDP4_MAX_TERMS ||
      desc->n_couplings < 1 || desc->n_couplings > TDDP4_MAX_COUPLINGS)
    return bail(fail(h, TDDP4_ERR_ARG, "model size out of range"));
  if (!(desc->t_hi > desc->t_lo)) return bail(fail(h, TDDP4_ERR_ARG, "empty decay-time window"));
  if (desc->use_resolution < 0 || desc->use_resolution > 2) return bail(fail(h, TDDP4_ERR_ARG, "use_resolution must be 0, 1 or 2"));
  h->res.assign(desc->res, desc->res + desc->n_res);
  h->terms.assign(desc->terms, desc->terms + desc->n_terms);
  h->t_lo = desc->t_lo; h->t_hi = desc->t_hi; h->use_resolution = desc->use_resolution;
  ModelTab &M = h->M;
  memset(&M, 0, sizeof M);
  M.n_kc = desc->n_couplings;
  M.m_parent = desc->m_parent;
  for (int i = 0; i < 4; ++i) M.m_final[i] = desc->m_final[i];
  M.r_res2 = desc->r_res * desc->r_res;
  M.r_parent2 = desc->r_parent * desc->r_parent;
  M.sysD = find_or_add_sys(M, 0xF);
  // terms sorted by coupling (stable), so that each column is a contiguous range
  std::vector<int> order(desc->n_terms);
  for (int k = 0; k < desc->n_terms; ++k) order[k] = k;
  std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return desc->terms[a].coupling < desc->terms[b].coupling; });
  for (int r = 0; r < desc->n_res; ++r)
    if (desc->res[r].L < 0 || desc->res[r].L > 2 || desc->res[r].lineshape < 0 || desc->res[r].lineshape > LS_CONSTANT ||
        !(desc->res[r].r >= 0.0))
      return bail(fail(h, TDDP4_ERR_ARG, "resonance %d: L must be 0, 1 or 2, lineshape 0 or 1, r >= 0", r));
  int pos = 0;
  for (int kap = 0; kap <= M.n_kc; ++kap) {
    M.col_begin[kap] = (int8_t)pos;
    while (kap < M.n_kc && pos < desc->n_terms && desc->terms[order[pos]].coupling == kap) ++pos;
  }
  if (pos != desc->n_terms) return bail(fail(h, TDDP4_ERR_ARG, "term coupling index out of range"));
  M.n_terms = desc->n_terms;
  for (int k = 0; k < M.n_terms; ++k) {
    const tddp4_term &t = desc->terms[order[k]];
    TermTab &tm = M.term[k];
    M.user_term[k] = (int8_t)order[k];
    unsigned seen = 0;
    for (int r = 0; r < 4; ++r) {
      if (t.perm[r] < 0 || t.perm[r] > 3) return bail(fail(h, TDDP4_ERR_ARG, "term %d: bad permutation", order[k]));
      seen |= 1u << t.perm[r];
      tm.perm[r] = (int8_t)t.perm[r];
    }
    if (seen != 0xF) return bail(fail(h, TDDP4_ERR_ARG, "term %d: perm is not a permutation", order[k]));
    if (t.spin_factor < SF_NONRES || t.spin_factor > SF_AP_D)
      return bail(fail(h, TDDP4_ERR_ARG, "term %d: unknown spin factor", order[k]));
    tm.sf = (int8_t)t.spin_factor;
    tm.LD = (int8_t)parent_L(t.spin_factor);
    tm.inst0 = tm.inst1 = -1;
    if (t.spin_factor == SF_NONRES) continue;
    for (int r = 0; r < 2; ++r)
      if (t.res[r] < 0 || t.res[r] >= desc->n_res) return bail(fail(h, TDDP4_ERR_ARG, "term %d: bad resonance index", order[k]));
    const int *pm = t.perm;
    InstTab a{}, b{};
    a.dres = b.dres = -1;
    if (t.spin_factor <= SF_VV_D) {
      a.res = (int8_t)t.res[0]; a.sys = (int8_t)find_or_add_sys(M, (1u << pm[0]) | (1u << pm[1])); a.sub = -1;
      a.ma = M.m_final[pm[0]]; a.mb = M.m_final[pm[1]];
      b.res = (int8_t)t.res[1]; b.sys = (int8_t)find_or_add_sys(M, (1u << pm[2]) | (1u << pm[3])); b.sub = -1;
      b.ma = M.m_final[pm[2]]; b.mb = M.m_final[pm[3]];
    } else {
      int sysV = find_or_add_sys(M, (1u << pm[0]) | (1u << pm[1]));
      a.res = (int8_t)t.res[0]; a.sys = (int8_t)find_or_add_sys(M, (1u << pm[0]) | (1u << pm[1]) | (1u << pm[2]));
      a.sub = (int8_t)sysV; a.dres = (int8_t)t.res[1]; a.ma = 0.0; a.mb = M.m_final[pm[2]];
      b.res = (int8_t)t.res[1]; b.sys = (int8_t)sysV; b.sub = -1; b.ma = M.m_final[pm[0]]; b.mb = M.m_final[pm[1]];
    }
    a.L = (int8_t)desc->res[a.res].L;
    b.L = (int8_t)desc->res[b.res].L;
    a.kind = (int8_t)desc->res[a.res].lineshape;
    b.kind = (int8_t)desc->res[b.res].lineshape;
    a.r2 = desc->res[a.res].r > 0.0 ? desc->res[a.res].r * desc->res[a.res].r : M.r_res2;
    b.r2 = desc->res[b.res].r > 0.0 ? desc->res[b.res].r * desc->res[b.res].r : M.r_res2;
    if (a.sys < 0 || b.sys < 0) return bail(fail(h, TDDP4_ERR_ARG, "too many particle systems"));
    int ia = find_or_add_inst(M, a), ib = find_or_add_inst(M, b);
    if (ia < 0 || ib < 0) return bail(fail(h, TDDP4_ERR_ARG, "too many lineshape instances"));
    tm.inst0 = (int8_t)ia; tm.inst1 = (int8_t)ib;
  }
  // renumber the particle systems so that those no lineshape reads (the four-body system, ...) come FIRST: the rows
  // the per-call kernels stream are then one contiguous range of every tile, and the bulk L2 prefetch can skip the rest
  {
    bool used[MAX_SYS] = {false};
    for (int j = 0; j < M.n_inst; ++j) used[M.inst[j].sys] = true;
    int remap[MAX_SYS], next = 0;
    for (int pass = 0; pass < 2; ++pass)
      for (int i = 0; i < M.n_sys; ++i)
        if (used[i] == (pass == 1)) remap[i] = next++;
    M.n_su = 0;
    for (int i = 0; i < M.n_sys; ++i) M.n_su += used[i] ? 1 : 0;
    uint8_t mask[MAX_SYS];
    for (int i = 0; i < M.n_sys; ++i) mask[remap[i]] = M.sys_mask[i];
    for (int i = 0; i < M.n_sys; ++i) M.sys_mask[i] = mask[i];
    M.sysD = remap[M.sysD];
    for (int j = 0; j < M.n_inst; ++j) {
      M.inst[j].sys = (int8_t)remap[M.inst[j].sys];
      if (M.inst[j].sub >= 0) M.inst[j].sub = (int8_t)remap[M.inst[j].sub];
    }
  }
  {   // flat tables of the per-call kernels (tables.h): padded to groups of 4, all entries 32-bit
    StreamTab &S = h->S;
    memset(&S, 0, sizeof S);
    // size class = load-batch sizes (GI, GT): the one with the fewest padded rows, the deeper batches on a tie
    static const int GI[3] = {4, 8, 12}, GT[3] = {4, 8, 16};
    int best = -1;
    for (int c = 0; c < 3; ++c) {
      int ni = (M.n_inst + GI[c] - 1) / GI[c] * GI[c], nt = (M.n_terms + GT[c] - 1) / GT[c] * GT[c];
      if (ni > MAX_INST || nt > MAX_TERMS) continue;
      if (best < 0 || ni + nt <= S.n_inst4 + S.n_terms4) { best = c; S.n_inst4 = ni; S.n_terms4 = nt; }
    }
    h->size_class = best;
    S.n_kc = M.n_kc;
    S.g_off = M.n_sys * 32; S.f_off = (M.n_sys + S.n_inst4) * 32; S.w_off = -1;
    S.skip = (M.n_sys - M.n_su) * 32;                    // leading rows nobody streams
    S.R = M.n_sys + S.n_inst4 + S.n_terms4;              // + 1 for a weighted event set, fixed at launch
    for (int j = 0; j < M.n_inst; ++j) S.inst_soff[j] = (uint32_t)M.inst[j].sys * 32;
    const uint32_t unit = (uint32_t)S.n_inst4 * 32;
    for (int k = 0; k < MAX_TERMS; ++k) { S.term_t0[k] = S.term_t1[k] = unit; }
    for (int kap = 0; kap < M.n_kc; ++kap)
      for (int k = M.col_begin[kap]; k < M.col_begin[kap + 1]; ++k) {
        const TermTab &tm = M.term[k];
        if (tm.inst0 >= 0) { S.term_t0[k] = (uint32_t)tm.inst0 * 32; S.term_t1[k] = (uint32_t)tm.inst1 * 32; }
        S.term_col[k] = (uint32_t)kap;
        S.term_last[k] = k == M.col_begin[kap + 1] - 1;
      }
  }
  if (h->use_resolution) fadd_coefficients(h->FT);
  h->mass.assign(desc->n_res, 0.0);
  h->width.assign(desc->n_res, 0.0);

  cudaError_t e = cudaGetDevice(&h->device);
  if (e != cudaSuccess) return bail(fail(h, TDDP4_ERR_CUDA, "cudaGetDevice: %s (no CPU fallback exists)", cudaGetErrorString(e)));
  cudaDeviceProp prop;
  e = cudaGetDeviceProperties(&prop, h->device);
  if (e != cudaSuccess) return bail(fail(h, TDDP4_ERR_CUDA, "cudaGetDeviceProperties: %s", cudaGetErrorString(e)));
  h->sm_count = prop.multiProcessorCount;
  e = cudaStreamCreateWithFlags(&h->stream, cudaStreamNonBlocking);
  if (e != cudaSuccess) return bail(fail(h, TDDP4_ERR_CUDA, "cudaStreamCreate: %s", cudaGetErrorString(e)));
  h->own_stream = true;
  int KC = M.n_kc;
  bool ok = cudaMalloc(&h->G, sizeof(double) * 2 * KC * KC) == cudaSuccess &&
            cudaMalloc(&h->ticket, sizeof(unsigned int) * MAX_TICKETS) == cudaSuccess &&
            cudaMalloc(&h->results, sizeof(double) * (N_SLOTS + 1) * SLOT_DOUBLES) == cudaSuccess &&
            cudaHostAlloc(&h->results_host, sizeof(double) * N_SLOTS * SLOT_DOUBLES, cudaHostAllocMapped) == cudaSuccess &&
            cudaHostGetDevicePointer((void **)&h->results_host_dev, h->results_host, 0) == cudaSuccess &&
            cudaHostAlloc(&h->grad_host, sizeof(double) * (GRAD_OFFSET + 4 * MAX_KC + 2), cudaHostAllocMapped) == cudaSuccess &&
            cudaHostGetDevicePointer((void **)&h->grad_host_dev, h->grad_host, 0) == cudaSuccess &&
            cudaMalloc(&h->gen_scalars, sizeof(unsigned long long) * 4) == cudaSuccess &&
            cudaMalloc(&h->tres_tab, sizeof(TresTable)) == cudaSuccess &&
            cudaMemset(h->ticket, 0, sizeof(unsigned int) * MAX_TICKETS) == cudaSuccess &&
            cudaMemset(h->G, 0, sizeof(double) * 2 * KC * KC) == cudaSuccess;
  if (ok) memset(h->results_host, 0, sizeof(double) * N_SLOTS * SLOT_DOUBLES);   // no stale sequence stamps from a recycled allocation
  for (int s = 0; ok && s < N_SLOTS; ++s) ok = cudaEventCreateWithFlags(&h->slot_event[s], cudaEventDisableTiming) == cudaSuccess;
  if (!ok) return bail(fail(h, TDDP4_ERR_CUDA, "allocation failed: %s", cudaGetErrorString(cudaGetLastError())));
  // kernels that need more than 48 KB of dynamic shared memory
  cudaFuncSetAttribute(gen_ratio_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gen_smem_bytes(MAX_SYS, MAX_INST));
  cudaFuncSetAttribute(kin_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(sizeof(double) * (16 + MAX_SYS + MAX_INST) * KIN_BLOCK));
  {   // shared memory of the per-call kernels: per-warp lineshape scratch (+ the X tile of the Gram kernel)
    int NB = (KC + 3) / 4;
    size_t limit = prop.sharedMemPerBlockOptin - 1024, sc = colnll_smem_bytes(h->S.n_inst4), sg = gram_smem_bytes(NB, h->S.n_inst4);
    if (sc > limit || sg > limit) return bail(fail(h, TDDP4_ERR_ARG, "model too large for the shared-memory scratch of the streaming kernels"));
    with_size_class(h->size_class, [&](auto ni, auto nt) {
      constexpr int NI = decltype(ni)::value, NT = decltype(nt)::value;
      cudaFuncSetAttribute(colnll_stream_kernel<true, false, NI, NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sc);
      cudaFuncSetAttribute(colnll_stream_kernel<false, false, NI, NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sc);
      cudaFuncSetAttribute(colnll_stream_kernel<false, true, NI, NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sc);
      if (NB == 1) cudaFuncSetAttribute(gram_stream_kernel<1, NI, NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sg);
      else if (NB == 2) cudaFuncSetAttribute(gram_stream_kernel<2, NI, NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sg);
      else if (NB == 3) cudaFuncSetAttribute(gram_stream_kernel<3, NI, NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sg);
      else cudaFuncSetAttribute(gram_stream_kernel<4, NI, NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sg);
      return 0;
    });
  }
  cudaFuncSetAttribute(terms_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(MAX_INST * COL_BLOCK * sizeof(double2)));
  switch (KC) {   // the gradient kernels' per-warp tiles (grad_kernels.cuh)
#define CASE(k) case k: cudaFuncSetAttribute(nll_grad_kernel<k, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)grad_smem_bytes<k>()); \
                        cudaFuncSetAttribute(nll_grad_kernel<k, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)grad_smem_bytes<k>()); \
                        cudaFuncSetAttribute(nll_grad_res_kernel<k>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)grad_smem_bytes<k>()); break;
    CASE(1) CASE(2) CASE(3) CASE(4) CASE(5) CASE(6) CASE(7) CASE(8) CASE(9) CASE(10) CASE(11) CASE(12)
    CASE(13) CASE(14) CASE(15) CASE(16)
#undef CASE
  }
  *out = h;
  return TDDP4_OK;
}

int tddp4_destroy(tddp4 *h) {
  if (!h) return TDDP4_OK;
  if (h->stream) cudaStreamSynchronize(h->stream);
  drain_profile(h);
  for (auto e : h->pool) cudaEventDestroy(e);
  free_set(h->set[0]);
  free_set(h->set[1]);
  cudaFree(h->G); cudaFree(h->partials); cudaFree(h->ticket); cudaFree(h->results); cudaFree(h->batch_res); cudaFree(h->tres_tab); cudaFree(h->staging);
  if (h->batch_res_host) cudaFreeHost(h->batch_res_host);
  if (h->results_host) cudaFreeHost(h->results_host);
  if (h->grad_host) cudaFreeHost(h->grad_host);
  cudaFree(h->gen_flags); cudaFree(h->gen_counts); cudaFree(h->gen_offs); cudaFree(h->gen_scalars);
  for (int s = 0; s < N_SLOTS; ++s)
    if (h->slot_event[s]) cudaEventDestroy(h->slot_event[s]);
  if (h->own_stream && h->stream) cudaStreamDestroy(h->stream);
  delete h;
  return TDDP4_OK;
}

int tddp4_set_stream(tddp4 *h, void *cuda_stream) {
  if (!h) return TDDP4_ERR_ARG;
  if (h->stream) CU(cudaStreamSynchronize(h->stream));
  if (h->own_stream) { cudaStreamDestroy(h->stream); h->own_stream = false; }
  h->stream = (cudaStream_t)cuda_stream;
  h->prev_kind = PREV_NONE;
  return TDDP4_OK;
}

int tddp4_load_events(tddp4 *h, int which, int64_t n, int64_t ld_in, const double *p4, const double *t,
                      const double *sigma_t, const double *weight, int on_device) {
  if (!h) return TDDP4_ERR_ARG;
  if (which < 0 || which > 1 || n < 0 || ld_in < n || (n > 0 && !p4)) return fail(h, TDDP4_ERR_ARG, "bad load_events argument");
  if (which == 0 && n > 0 && !t && h->use_resolution != 2) return fail(h, TDDP4_ERR_ARG, "the data sample needs decay times");
  if (which == 0 && n > 0 && h->use_resolution == 1 && !sigma_t)
    return fail(h, TDDP4_ERR_ARG, "use_resolution = 1: the data sample needs per-event sigma_t");
  CU(cudaStreamSynchronize(h->stream));
  h->prev_kind = PREV_NONE;
  if (which == 0) h->store_mask = 0xFFFFFFFFu;
  EventSet &e = h->set[which];
  const ModelTab &M = h->M;
  const int R_new = h->S.R + (weight && n > 0 ? 1 : 0);
  // a reload of the same shape (same n, same optional rows) keeps every allocation: the padding rows, the ragged tail
  // and the columns of couplings without chains are still zero, everything else is rewritten below
  const bool reuse = e.loaded && e.n == n && e.R == R_new && n > 0 && (e.t != nullptr) == (t != nullptr) &&
                     (e.sigma_t != nullptr) == (sigma_t != nullptr) && (e.w != nullptr) == (weight != nullptr);
  if (!reuse) {
    free_set(e);
    e.n = n;
    e.ld = std::max<int64_t>(32, (n + 31) / 32 * 32);   // rows start 256-byte aligned
    e.R = R_new;
    CU(cudaMalloc(&e.cache, sizeof(double) * e.R * e.ld));
    CU(cudaMemsetAsync(e.cache, 0, sizeof(double) * e.R * e.ld, h->stream));   // padding rows and the ragged tail stay zero
    if (which == 0) {   // the normalisation sample keeps no columns; a coupling without chains keeps its zero column
      CU(cudaMalloc(&e.a, sizeof(double2) * M.n_kc * e.ld));
      CU(cudaMemsetAsync(e.a, 0, sizeof(double2) * M.n_kc * e.ld, h->stream));
      if (h->use_resolution) CU(cudaMalloc(&e.tr, sizeof(double) * 8 * e.ld));
    }
  }
  e.tres_valid = e.tresg_valid = false;
  e.tres_parts = 3;
  const CacheRows cr{e.R, M.n_sys, M.n_sys + h->S.n_inst4};
  cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  auto copy_vec = [&](double **dst, const double *src) -> cudaError_t {
    if (!src || n == 0) return cudaSuccess;
    if (!*dst) {
      cudaError_t e_ = cudaMalloc(dst, sizeof(double) * e.ld);
      if (e_ != cudaSuccess) return e_;
    }
    return cudaMemcpyAsync(*dst, src, sizeof(double) * n, kind, h->stream);
  };
  CU(copy_vec(&e.t, t));
  CU(copy_vec(&e.sigma_t, sigma_t));
  CU(copy_vec(&e.w, weight));
  if (n > 0) {
    const double *dp4 = p4;
    int64_t ld_dev = ld_in;
    if (!on_device) {   // host input goes through a staging buffer the handle keeps (grow-only)
      if ((size_t)(16 * n) > h->staging_cap) {
        cudaFree(h->staging);
        h->staging = nullptr; h->staging_cap = 0;
        CU(cudaMalloc(&h->staging, sizeof(double) * 16 * n));
        h->staging_cap = (size_t)(16 * n);
      }
      CU(cudaMemcpy2DAsync(h->staging, sizeof(double) * n, p4, sizeof(double) * ld_in, sizeof(double) * n, 16,
                           cudaMemcpyHostToDevice, h->stream));
      dp4 = h->staging;
      ld_dev = n;
    }
    int grid = (int)((n + KIN_BLOCK - 1) / KIN_BLOCK);
    size_t smem = sizeof(double) * (16 + M.n_sys + M.n_inst) * KIN_BLOCK;
    {
      Prof p(h, TDDP4_K_KIN, (double)n * 8.0 * (16 + M.n_sys + M.n_inst + M.n_terms));
      kin_kernel<<<grid, KIN_BLOCK, smem, h->stream>>>(M, dp4, ld_dev, n, e.cache, cr);
    }
    CU(cudaGetLastError());
    if (e.w) {   // the weights travel with the rows they multiply
      row_scatter_kernel<<<(int)((n + 255) / 256), 256, 0, h->stream>>>(e.cache, e.R, e.R - 1, n, e.w);
      ++h->launches;
      CU(cudaGetLastError());
    }
    double st[6] = {0};
    if (e.t) {
      stat_kernel<<<1, 1024, 0, h->stream>>>(e.t, n, h->results);   // slot 0 as scratch
      ++h->launches;
      if (e.sigma_t) { stat_kernel<<<1, 1024, 0, h->stream>>>(e.sigma_t, n, h->results + 3); ++h->launches; }
      CU(cudaMemcpyAsync(st, h->results, 6 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    }
    CU(cudaStreamSynchronize(h->stream));        // the one synchronisation of a load: the caller's buffers are free again
    if (e.t) {
      e.sum_t = st[0];
      e.t_max = st[1];
      if (e.sigma_t) { e.sig_lo = st[5]; e.sig_hi = st[4]; }   // sigma_t > 0: max |.| = max
    }
  }
  e.cols_dirty = true;
  e.loaded = true;
  if (which == 1) { h->gram_valid = false; h->gram_overridden = false; }
  return TDDP4_OK;
}

int tddp4_set_params(tddp4 *h, const double *c, const double *cbar, const double *mass_width, double x, double y,
                     double tau) {
  if (!h || !c || !cbar || (h->res.size() && !mass_width)) return fail(h, TDDP4_ERR_ARG, "null parameter block");
  if (!(tau > 0.0) || !(std::fabs(y) < 1.0)) return fail(h, TDDP4_ERR_ARG, "need tau > 0 and |y| < 1");
  const ModelTab &M = h->M;
  LineParams lp{};
  for (int j = 0; j < MAX_INST; ++j) { lp.m0sq[j] = -1.0; lp.gam[j] = 0.0; }   // padded instances: finite, unused
  int nres = (int)h->res.size();
  for (int j = 0; j < M.n_inst; ++j) {
    const InstTab &in = M.inst[j];
    double m0 = mass_width[2 * in.res], g0 = mass_width[2 * in.res + 1];
    double ma0 = in.dres >= 0 ? mass_width[2 * in.dres] : in.ma;
    lp.m0sq[j] = m0 * m0;
    if (in.kind == LS_CONSTANT) {                       // constant width: shape row g = 1, m0 Gamma = m0 Gamma0
      if (!(m0 > 0.0) || !(g0 > 0.0)) return fail(h, TDDP4_ERR_DOMAIN, "resonance %d: mass and width must be positive", (int)in.res);
      lp.gam[j] = m0 * g0;
      continue;
    }
    if (!(m0 > ma0 + in.mb) || !(g0 > 0.0))
      return fail(h, TDDP4_ERR_DOMAIN, "resonance %d: pole mass %.6g below its decay threshold %.6g (or width <= 0)",
                  (int)in.res, m0, ma0 + in.mb);
    double q0 = host_breakup(m0, ma0, in.mb);
    double z0 = q0 * q0 * in.r2;
    lp.gam[j] = m0 * m0 * g0 / (std::pow(q0, 2 * in.L + 1) * host_barrier2(in.L, z0));
  }
  bool dirty = !h->have_params;                       // any lineshape constant moved: columns and Gram are stale
  bool moved[MAX_INST] = {false};
  for (int j = 0; j < M.n_inst; ++j)
    if (lp.m0sq[j] != h->LP.m0sq[j] || lp.gam[j] != h->LP.gam[j]) dirty = moved[j] = true;
  if (!h->have_params) h->store_mask = 0xFFFFFFFFu;
  for (int kap = 0; kap < M.n_kc; ++kap)              // which stored columns that makes stale (accumulates until rebuilt)
    for (int k = M.col_begin[kap]; k < M.col_begin[kap + 1]; ++k)
      if (M.term[k].inst0 >= 0 && (moved[M.term[k].inst0] || moved[M.term[k].inst1])) h->store_mask |= 1u << kap;
  h->LP = lp;
  for (int r = 0; r < nres; ++r) { h->mass[r] = mass_width[2 * r]; h->width[r] = mass_width[2 * r + 1]; }
  RateParams &R = h->RP;
  for (int k = 0; k < M.n_kc; ++k) {
    R.c[k][0] = c[2 * k]; R.c[k][1] = c[2 * k + 1];
    R.cbar[k][0] = cbar[2 * k]; R.cbar[k][1] = cbar[2 * k + 1];
  }
  if (R.x != x || R.y != y || R.Gamma != 1.0 / tau || !h->have_params) {
    h->set[0].tres_valid = h->set[0].tresg_valid = false;
    if (R.Gamma != 1.0 / tau || !h->have_params) h->set[0].tres_parts = 3;
    if (R.y != y) h->set[0].tres_parts |= 1;
    if (R.x != x) h->set[0].tres_parts |= 2;
  }
  R.x = x; R.y = y; R.Gamma = 1.0 / tau;
  R.t_lo = h->t_lo; R.t_hi = h->t_hi; R.use_resolution = h->use_resolution;
  time_integrals(x, y, R.Gamma, h->t_lo, h->t_hi, R.T);
  if (dirty) {
    h->set[0].cols_dirty = true;
    h->gram_valid = false;
    h->gram_overridden = false;
  }
  h->have_params = true;
  return TDDP4_OK;
}

int tddp4_nll_async(tddp4 *h, int slot) {
  if (!h || slot < 0 || slot >= N_SLOTS) return fail(h, TDDP4_ERR_ARG, "bad slot");
  return enqueue_nll_slot(h, slot, nullptr);
}

int tddp4_nll_result(tddp4 *h, int slot, double *nll_out) {
  if (!h || slot < 0 || slot >= N_SLOTS || !nll_out) return fail(h, TDDP4_ERR_ARG, "bad slot");
  if (!h->slot_used[slot]) return fail(h, TDDP4_ERR_STATE, "slot %d holds no evaluation", slot);
  int wrc = wait_slot(h, slot);
  if (wrc) return wrc;
  const double *r = h->results_host + (size_t)slot * SLOT_DOUBLES;
  *nll_out = r[3];
  if (r[4] > 0.0 || !std::isfinite(r[3])) {
    *nll_out = INFINITY;
    return fail(h, TDDP4_ERR_NONFINITE, "%g events with non-positive or non-finite rate (N = %g)", r[4], r[2]);
  }
  return TDDP4_OK;
}

int tddp4_nll(tddp4 *h, double *nll_out, double *prob_out) {
  if (!h || !nll_out) return fail(h, TDDP4_ERR_ARG, "null argument");
  int rc = enqueue_nll_slot(h, 0, prob_out);
  if (rc) return rc;
  return tddp4_nll_result(h, 0, nll_out);
}

int tddp4_nll_grad(tddp4 *h, double *nll_out, double *grad_out) {
  if (!h || !nll_out || !grad_out) return fail(h, TDDP4_ERR_ARG, "null argument");
  if (!h->have_params) return fail(h, TDDP4_ERR_STATE, "tddp4_set_params has not been called");
  EventSet &d = h->set[0];
  if (!d.loaded) return fail(h, TDDP4_ERR_STATE, "data sample not loaded");
  int rc;
  if (d.cols_dirty || !h->gram_valid || (h->use_resolution && !d.tres_valid)) {   // columns, Gram matrix, time rows up to date
    rc = enqueue_nll(h, h->results + (size_t)N_SLOTS * SLOT_DOUBLES, nullptr);
    if (rc) return rc;
  }
  double inv_n = h->gram_n > 0 ? 1.0 / (double)h->gram_n : 0.0;
  const RateParams &R = h->RP;
  bool small = std::fabs(R.y) * R.Gamma * d.t_max < 0.25 && std::fabs(R.x) * R.Gamma * d.t_max < 0.25;
  if (h->use_resolution && !d.tresg_valid && d.n > 0) {   // derivative rows: rebuilt when x, y, tau or the sample changed
    if (!d.trg) CU(cudaMalloc(&d.trg, sizeof(double) * 8 * d.ld));
    int grid = (int)((d.n + TRES_BLOCK - 1) / TRES_BLOCK);
    if (h->use_resolution == 2) {          // time-integrated: constant derivative rows (dT1/dx, dT3/dx, dT0/dy, dT2/dy) twice
      GradParams gp = time_integral_derivatives(R.x, R.y, R.Gamma, h->t_lo, h->t_hi);
      Row8 v;
      v.v[0] = v.v[4] = gp.dT1dx; v.v[1] = v.v[5] = gp.dT3dx; v.v[2] = v.v[6] = gp.dT0dy; v.v[3] = v.v[7] = gp.dT2dy;
      Prof p(h, TDDP4_K_TRES, (double)d.n * 64.0);
      fill_rows_kernel<<<(int)((d.n + 255) / 256), 256, 0, h->stream>>>(d.trg, d.ld, d.n, v);
    } else {
      Prof p(h, TDDP4_K_TRES, (double)d.n * 80.0);
      tres_grad_kernel<<<grid, TRES_BLOCK, 0, h->stream>>>(h->FT, d.t, d.sigma_t, d.n, R.x, R.y, R.Gamma, h->t_lo, h->t_hi, d.trg, d.ld);
    }
    CU(cudaGetLastError());
    d.tresg_valid = true;
  }
  switch (h->M.n_kc) {
#define CASE(k) case k: rc = h->use_resolution ? launch_nll_grad_res<k>(h, d, inv_n) : launch_nll_grad<k>(h, d, inv_n, small); break;
    CASE(1) CASE(2) CASE(3) CASE(4) CASE(5) CASE(6) CASE(7) CASE(8) CASE(9) CASE(10) CASE(11) CASE(12)
    CASE(13) CASE(14) CASE(15) CASE(16)
#undef CASE
    default: return fail(h, TDDP4_ERR_ARG, "unsupported number of couplings %d", h->M.n_kc);
  }
  if (rc) return rc;
  CU(cudaGetLastError());
  h->prev_kind = PREV_NONE;
  CU(cudaStreamSynchronize(h->stream));
  const double *r = h->grad_host;
  const int na = 4 * h->M.n_kc + 2;
  memcpy(grad_out, r + GRAD_OFFSET, sizeof(double) * na);
  *nll_out = r[3];
  if (r[4] > 0.0 || !std::isfinite(r[3])) {
    *nll_out = INFINITY;
    return fail(h, TDDP4_ERR_NONFINITE, "%g events with non-positive or non-finite rate (N = %g)", r[4], r[2]);
  }
  return TDDP4_OK;
}

int tddp4_nll_parts(tddp4 *h, int slot, double out[5]) {
  if (!h || slot < 0 || slot >= N_SLOTS || !out) return fail(h, TDDP4_ERR_ARG, "bad slot");
  if (!h->slot_used[slot]) return fail(h, TDDP4_ERR_STATE, "slot %d holds no evaluation", slot);
  int wrc = wait_slot(h, slot);
  if (wrc) return wrc;
  memcpy(out, h->results_host + (size_t)slot * SLOT_DOUBLES, 5 * sizeof(double));
  return TDDP4_OK;
}

int tddp4_param_stride(const tddp4 *h) { return h ? 4 * h->M.n_kc + 2 * (int)h->res.size() + 3 : TDDP4_ERR_ARG; }

int tddp4_nll_batch(tddp4 *h, int64_t n_points, const double *params, double *nll_out, int *status_out) {
  if (!h || n_points < 0 || (n_points > 0 && (!params || !nll_out))) return fail(h, TDDP4_ERR_ARG, "bad argument");
  if (n_points == 0) return TDDP4_OK;
  if (n_points > h->batch_cap) {
    cudaFree(h->batch_res);
    if (h->batch_res_host) cudaFreeHost(h->batch_res_host);
    h->batch_res = nullptr; h->batch_res_host = nullptr; h->batch_cap = 0;
    CU(cudaMalloc(&h->batch_res, sizeof(double) * SLOT_DOUBLES * n_points));
    CU(cudaMallocHost(&h->batch_res_host, sizeof(double) * SLOT_DOUBLES * n_points));
    h->batch_cap = n_points;
  }
  const int KC = h->M.n_kc, nres = (int)h->res.size(), stride = 4 * KC + 2 * nres + 3;
  int first_err = TDDP4_OK;
  std::vector<int> st((size_t)n_points, TDDP4_OK);
  for (int64_t i = 0; i < n_points; ++i) {
    const double *p = params + i * stride;
    const double *tail = p + 4 * KC + 2 * nres;
    int rc = tddp4_set_params(h, p, p + 2 * KC, p + 4 * KC, tail[0], tail[1], tail[2]);
    if (!rc) rc = enqueue_nll(h, h->batch_res + i * SLOT_DOUBLES, nullptr);
    st[i] = rc;
    if (rc == TDDP4_ERR_CUDA) return rc;
  }
  CU(cudaMemcpyAsync(h->batch_res_host, h->batch_res, sizeof(double) * SLOT_DOUBLES * n_points, cudaMemcpyDeviceToHost,
                     h->stream));
  CU(cudaStreamSynchronize(h->stream));
  for (int64_t i = 0; i < n_points; ++i) {
    const double *r = h->batch_res_host + i * SLOT_DOUBLES;
    if (st[i] == TDDP4_OK) {
      nll_out[i] = r[3];
      if (r[4] > 0.0 || !std::isfinite(r[3])) {
        nll_out[i] = INFINITY;
        st[i] = fail(h, TDDP4_ERR_NONFINITE, "point %lld: %g events with non-positive or non-finite rate (N = %g)",
                     (long long)i, r[4], r[2]);
      }
    } else {
      nll_out[i] = std::numeric_limits<double>::quiet_NaN();
    }
    if (status_out) status_out[i] = st[i];
    if (st[i] && !first_err) first_err = st[i];
  }
  return first_err;
}

int tddp4_gram(tddp4 *h, double *G_sum, int64_t *n_norm) {
  if (!h || !G_sum || !n_norm) return fail(h, TDDP4_ERR_ARG, "null argument");
  if (!h->have_params) return fail(h, TDDP4_ERR_STATE, "tddp4_set_params has not been called");
  if (h->gram_overridden) { h->gram_valid = false; h->gram_overridden = false; }
  int rc = ensure_gram(h);
  if (rc) return rc;
  int KC = h->M.n_kc;
  CU(cudaMemcpyAsync(G_sum, h->G, sizeof(double) * 2 * KC * KC, cudaMemcpyDeviceToHost, h->stream));
  CU(cudaStreamSynchronize(h->stream));
  *n_norm = h->gram_n;
  return TDDP4_OK;
}

int tddp4_gram_override(tddp4 *h, const double *G_sum, int64_t n_norm) {
  if (!h || !G_sum || n_norm <= 0) return fail(h, TDDP4_ERR_ARG, "bad argument");
  int KC = h->M.n_kc;
  CU(cudaMemcpyAsync(h->G, G_sum, sizeof(double) * 2 * KC * KC, cudaMemcpyHostToDevice, h->stream));
  CU(cudaStreamSynchronize(h->stream));
  h->gram_valid = true;
  h->gram_overridden = true;
  h->gram_n = n_norm;
  return TDDP4_OK;
}

int tddp4_gram_state(const tddp4 *h, int *valid, int *overridden) {
  if (!h) return TDDP4_ERR_ARG;
  if (valid) *valid = h->gram_valid ? 1 : 0;
  if (overridden) *overridden = h->gram_overridden ? 1 : 0;
  return TDDP4_OK;
}

int tddp4_gram_enqueue(tddp4 *h, double *G_dev) {
  if (!h || !G_dev) return fail(h, TDDP4_ERR_ARG, "null argument");
  if (!h->have_params) return fail(h, TDDP4_ERR_STATE, "tddp4_set_params has not been called");
  if (h->gram_overridden) { h->gram_valid = false; h->gram_overridden = false; }
  int rc = ensure_gram(h);
  if (rc) return rc;
  const int len = 2 * h->M.n_kc * h->M.n_kc;
  CU(cudaMemcpyAsync(G_dev, h->G, sizeof(double) * len, cudaMemcpyDeviceToDevice, h->stream));
  append_count_kernel<<<1, 32, 0, h->stream>>>(G_dev + len, (double)h->gram_n);
  ++h->launches;
  CU(cudaGetLastError());
  h->prev_kind = PREV_NONE;
  return TDDP4_OK;
}

int tddp4_gram_reduce(tddp4 *h, const double *gathered_dev, int world, int64_t n_norm_total) {
  if (!h || !gathered_dev || world < 1 || n_norm_total <= 0) return fail(h, TDDP4_ERR_ARG, "bad argument");
  const int len = 2 * h->M.n_kc * h->M.n_kc;
  gram_reduce_kernel<<<1, 256, 0, h->stream>>>(gathered_dev, world, len + 1, len, h->G);
  ++h->launches;
  CU(cudaGetLastError());
  h->gram_valid = true;
  h->gram_overridden = true;
  h->gram_n = n_norm_total;
  h->prev_kind = PREV_NONE;
  return TDDP4_OK;
}

int tddp4_nll_enqueue(tddp4 *h, double *result_dev) {
  if (!h || !result_dev) return fail(h, TDDP4_ERR_ARG, "null argument");
  int rc = enqueue_nll(h, result_dev, nullptr);
  h->prev_kind = PREV_NONE;      // the caller's collective follows on the stream: the next kernel waits early
  return rc;
}

int tddp4_fp64_peak(tddp4 *h, double *inst_per_s) {
  if (!h || !inst_per_s) return fail(h, TDDP4_ERR_ARG, "null argument");
  const int grid = h->sm_count * 4, iters = 256;
  cudaEvent_t a, b;
  CU(cudaEventCreate(&a));
  CU(cudaEventCreate(&b));
  double best = 0.0;
  for (int rep = 0; rep < 4; ++rep) {      // the first repetition warms up
    CU(cudaEventRecord(a, h->stream));
    fp64_peak_kernel<<<grid, 256, 0, h->stream>>>(h->results, 1.0000001, 1e-9, iters);
    CU(cudaEventRecord(b, h->stream));
    CU(cudaEventSynchronize(b));
    float ms = 0.f;
    CU(cudaEventElapsedTime(&ms, a, b));
    double rate = (double)grid * 256.0 * 8.0 * 16.0 * iters / (ms * 1e-3);
    if (rep > 0 && rate > best) best = rate;
  }
  h->launches += 4;
  cudaEventDestroy(a);
  cudaEventDestroy(b);
  h->prev_kind = PREV_NONE;
  *inst_per_s = best;
  return TDDP4_OK;
}

int tddp4_norm(tddp4 *h, double *norm_out) {
  if (!h || !norm_out) return fail(h, TDDP4_ERR_ARG, "null argument");
  if (!h->have_params) return fail(h, TDDP4_ERR_STATE, "tddp4_set_params has not been called");
  int rc = ensure_gram(h);
  if (rc) return rc;
  int KC = h->M.n_kc;
  std::vector<double> G(2 * KC * KC);
  CU(cudaMemcpyAsync(G.data(), h->G, sizeof(double) * G.size(), cudaMemcpyDeviceToHost, h->stream));
  CU(cudaStreamSynchronize(h->stream));
  // same contraction as norm_from_gram() in the kernels, on the host copy
  const RateParams &R = h->RP;
  double inv_n = 1.0 / (double)h->gram_n, nAA = 0, nBB = 0, xr = 0, xi = 0;
  for (int k = 0; k < KC; ++k)
    for (int l = 0; l < KC; ++l) {
      double gr = G[(k * KC + l) * 2] * inv_n, gi = G[(k * KC + l) * 2 + 1] * inv_n;
      double pr = R.c[k][0] * R.c[l][0] + R.c[k][1] * R.c[l][1], pi = R.c[k][1] * R.c[l][0] - R.c[k][0] * R.c[l][1];
      nAA += pr * gr - pi * gi;
      pr = R.cbar[k][0] * R.cbar[l][0] + R.cbar[k][1] * R.cbar[l][1];
      pi = R.cbar[k][1] * R.cbar[l][0] - R.cbar[k][0] * R.cbar[l][1];
      nBB += pr * gr - pi * gi;
      pr = R.c[k][0] * R.cbar[l][0] + R.c[k][1] * R.cbar[l][1];
      pi = R.c[k][1] * R.cbar[l][0] - R.c[k][0] * R.cbar[l][1];
      xr += pr * gr - pi * gi;
      xi += pr * gi + pi * gr;
    }
  *norm_out = R.T[0] * (nAA + nBB) + R.T[1] * (nAA - nBB) - 2.0 * R.T[2] * xr - 2.0 * R.T[3] * xi;
  return TDDP4_OK;
}

// ---- generation ---------------------------------------------------------------------------------------
static int ensure_gen(tddp4 *h, int64_t n) {
  if (n <= h->gen_cap) return TDDP4_OK;
  cudaFree(h->gen_flags); cudaFree(h->gen_counts); cudaFree(h->gen_offs);
  h->gen_flags = nullptr; h->gen_counts = nullptr; h->gen_offs = nullptr; h->gen_cap = 0;
  int64_t blocks = (n + GEN_BLOCK - 1) / GEN_BLOCK;
  CU(cudaMalloc(&h->gen_flags, sizeof(uint32_t) * blocks * (GEN_BLOCK / 32)));
  CU(cudaMalloc(&h->gen_counts, sizeof(uint32_t) * blocks));
  CU(cudaMalloc(&h->gen_offs, sizeof(unsigned long long) * (blocks + 1)));
  h->gen_cap = n;
  return TDDP4_OK;
}

static int launch_ratio(tddp4 *h, uint64_t seed, uint32_t stream_id, uint64_t first, int64_t n, int mode, double env, int from_pilot,
                        double *p4, double *t, double *w, double *ratio, double *u) {
  int grid = (int)((n + GEN_BLOCK - 1) / GEN_BLOCK);
  {
    Prof p(h, TDDP4_K_GEN_RATIO);
    gen_ratio_kernel<<<grid, GEN_BLOCK, gen_smem_bytes(h->M.n_sys, h->M.n_inst), h->stream>>>(
        h->M, h->LP, h->RP, 1.0 / h->RP.Gamma, seed, stream_id, first, n, mode, env, from_pilot, p4, t, w, ratio, u,
        h->gen_scalars, h->gen_flags, h->gen_counts, h->gen_scalars + 1);
  }
  CU(cudaGetLastError());
  return TDDP4_OK;
}

int tddp4_candidates(tddp4 *h, uint64_t seed, uint32_t stream_id, int64_t first, int64_t n, double *out_p4,
                     double *out_t, double *out_w, double *out_ratio, double *out_u) {
  if (!h || n < 0 || first < 0) return fail(h, TDDP4_ERR_ARG, "bad argument");
  if (!h->have_params) return fail(h, TDDP4_ERR_STATE, "tddp4_set_params has not been called");
  if (n == 0) return TDDP4_OK;
  int rc = launch_ratio(h, seed, stream_id, (uint64_t)first, n, 0, 0.0, 0, out_p4, out_t, out_w, out_ratio, out_u);
  if (rc) return rc;
  CU(cudaStreamSynchronize(h->stream));
  return TDDP4_OK;
}

int tddp4_generate(tddp4 *h, uint64_t seed, uint32_t stream_id, int64_t first, int64_t n_candidates, int64_t n_pilot,
                   double envelope_scale, int64_t capacity, double *out_p4, double *out_t, int64_t *out_index,
                   int64_t *n_accepted, int64_t *n_overflow, double *envelope_out) {
  if (!h || n_candidates < 0 || n_pilot < 0 || capacity < 0 || first < 0 || !n_accepted || !n_overflow || !envelope_out)
    return fail(h, TDDP4_ERR_ARG, "bad argument");
  if (!h->have_params) return fail(h, TDDP4_ERR_STATE, "tddp4_set_params has not been called");
  const int64_t CHUNK = (int64_t)1 << 25;
  int rc = ensure_gen(h, std::min<int64_t>(std::max<int64_t>(n_candidates, n_pilot), CHUNK));
  if (rc) return rc;
  // device scalars: [0] pilot maximum (bit pattern), [1] overflow count, [2] running number of accepted candidates.
  // Everything is enqueued without a host round trip: the envelope is read by the ratio kernel from [0], the output
  // offsets of a chunk continue from [2]; one copy at the end brings the three words back.
  CU(cudaMemsetAsync(h->gen_scalars, 0, 3 * sizeof(unsigned long long), h->stream));
  const int from_pilot = n_pilot > 0;
  for (int64_t f = 0; f < n_pilot; f += CHUNK) {   // G5: exact, order-independent maximum over the pilot
    rc = launch_ratio(h, seed, stream_id, (uint64_t)f, std::min(CHUNK, n_pilot - f), 1, 0.0, 0, nullptr, nullptr, nullptr, nullptr, nullptr);
    if (rc) return rc;
  }
  for (int64_t f = 0; f < n_candidates; f += CHUNK) {   // G6
    int64_t n = std::min(CHUNK, n_candidates - f);
    int64_t blocks = (n + GEN_BLOCK - 1) / GEN_BLOCK;
    rc = launch_ratio(h, seed, stream_id, (uint64_t)(first + f), n, 2, envelope_scale, from_pilot, nullptr, nullptr, nullptr, nullptr, nullptr);
    if (rc) return rc;
    scan_kernel<<<1, 1024, 0, h->stream>>>(h->gen_counts, blocks, h->gen_offs, h->gen_scalars + 2);
    ++h->launches;
    CU(cudaGetLastError());
    {
      Prof p(h, TDDP4_K_GEN_EMIT);
      gen_emit_kernel<<<(int)((n + EMIT_SPAN - 1) / EMIT_SPAN), EMIT_BLOCK, 0, h->stream>>>(h->M, 1.0 / h->RP.Gamma, seed, stream_id,
                                                                                         (uint64_t)(first + f), n, h->gen_flags, h->gen_offs,
                                                                                         capacity, out_p4, out_t, out_index);
    }
    CU(cudaGetLastError());
  }
  unsigned long long sc[3] = {0, 0, 0};
  CU(cudaMemcpyAsync(sc, h->gen_scalars, sizeof sc, cudaMemcpyDeviceToHost, h->stream));
  CU(cudaStreamSynchronize(h->stream));
  double mx;
  memcpy(&mx, &sc[0], sizeof mx);
  const int64_t total = (int64_t)sc[2];
  *n_accepted = total;
  *n_overflow = (int64_t)sc[1];
  *envelope_out = from_pilot ? envelope_scale * mx : envelope_scale;
  if (total > capacity) return fail(h, TDDP4_ERR_CAPACITY, "%lld accepted events exceed capacity %lld", (long long)total, (long long)capacity);
  return TDDP4_OK;
}

int tddp4_weight_bound(const tddp4 *h, double *bound_out) {
  if (!h || !bound_out) return TDDP4_ERR_ARG;
  const double *m = h->M.m_final;
  double M = h->M.m_parent;
  *bound_out = host_breakup(M, m[0] + m[1] + m[2], m[3]) * host_breakup(M - m[3], m[0] + m[1], m[2]) *
               host_breakup(M - m[2] - m[3], m[0], m[1]);
  return TDDP4_OK;
}

// ---- validation projections ----------------------------------------------------------------------------
int tddp4_project(tddp4 *h, int64_t n, int64_t ld, const double *p4, int n_bins, const double *ranges, int64_t *hist_out,
                  double *values_dev) {
  if (!h || n < 0 || ld < n || (n > 0 && !p4) || n_bins < 1 || n_bins > PROJ_MAX_BINS || !ranges || !hist_out)
    return fail(h, TDDP4_ERR_ARG, "bad tddp4_project argument");
  ProjRanges R;
  for (int k = 0; k < 5; ++k) {
    if (!(ranges[2 * k + 1] > ranges[2 * k])) return fail(h, TDDP4_ERR_ARG, "empty histogram range %d", k);
    R.lo[k] = ranges[2 * k]; R.hi[k] = ranges[2 * k + 1]; R.inv_width[k] = 1.0 / (ranges[2 * k + 1] - ranges[2 * k]);
  }
  unsigned long long *hist = nullptr;
  CU(cudaMalloc(&hist, sizeof(unsigned long long) * 5 * n_bins));
  CU(cudaMemsetAsync(hist, 0, sizeof(unsigned long long) * 5 * n_bins, h->stream));
  if (n > 0) {
    int grid = (int)std::min<int64_t>((n + PROJ_BLOCK - 1) / PROJ_BLOCK, (int64_t)h->sm_count * 8);
    project_kernel<<<grid, PROJ_BLOCK, 0, h->stream>>>(p4, ld, n, n_bins, R, hist, values_dev);
    ++h->launches;
  }
  cudaError_t e1 = cudaGetLastError();
  cudaError_t e2 = cudaMemcpyAsync(hist_out, hist, sizeof(unsigned long long) * 5 * n_bins, cudaMemcpyDeviceToHost, h->stream);
  cudaError_t e3 = cudaStreamSynchronize(h->stream);
  cudaFree(hist);
  h->prev_kind = PREV_NONE;
  CU(e1); CU(e2); CU(e3);
  return TDDP4_OK;
}

// ---- inspection ---------------------------------------------------------------------------------------
int tddp4_get(tddp4 *h, int which, int what, double *out) {
  if (!h || which < 0 || which > 1 || !out) return fail(h, TDDP4_ERR_ARG, "bad argument");
  EventSet &e = h->set[which];
  if (!e.loaded) return fail(h, TDDP4_ERR_STATE, "event set %d not loaded", which);
  const ModelTab &M = h->M;
  auto rows = [&](const double *src, int nrows, size_t elem) -> int {
    CU(cudaMemcpy2DAsync(out, elem * e.n, src, elem * e.ld, elem * e.n, nrows, cudaMemcpyDeviceToDevice, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    return TDDP4_OK;
  };
  const CacheRows cr{e.R, M.n_sys, M.n_sys + h->S.n_inst4};
  auto cache_rows = [&](int row0, int nrows, const int8_t *dst_row) -> int {   // tile-major rows -> plain [nrows][n]
    for (int r = 0; r < nrows && e.n > 0; ++r) {
      row_gather_kernel<<<(int)((e.n + 255) / 256), 256, 0, h->stream>>>(e.cache, e.R, row0 + r, e.n,
                                                                      out + (int64_t)(dst_row ? dst_row[r] : r) * e.n);
      ++h->launches;
    }
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(h->stream));
    return TDDP4_OK;
  };
  switch (what) {
    case TDDP4_GET_S: return cache_rows(0, M.n_sys, nullptr);
    case TDDP4_GET_SHAPE: return cache_rows(cr.g_row0, M.n_inst, nullptr);
    case TDDP4_GET_STATIC: return cache_rows(cr.f_row0, M.n_terms, M.user_term);
    case TDDP4_GET_COLUMNS: {
      if (which != 0) return fail(h, TDDP4_ERR_ARG, "the normalisation sample keeps no coupling columns");
      if (!h->have_params) return fail(h, TDDP4_ERR_STATE, "tddp4_set_params has not been called");
      if (e.cols_dirty && e.n > 0) {                   // rebuild through the fused kernel; its NLL goes to a scratch slot
        int rc = enqueue_columns_only(h);
        if (rc) return rc;
      }
      return rows(reinterpret_cast<const double *>(e.a), M.n_kc, sizeof(double2));
    }
    case TDDP4_GET_TERMS: {
      if (!h->have_params) return fail(h, TDDP4_ERR_STATE, "tddp4_set_params has not been called");
      if (e.n == 0) return TDDP4_OK;
      int grid = (int)((e.n + COL_BLOCK - 1) / COL_BLOCK);
      size_t smem = (size_t)std::max(1, M.n_inst) * COL_BLOCK * sizeof(double2);
      terms_kernel<<<grid, COL_BLOCK, smem, h->stream>>>(M, h->LP, e.cache, cr, e.n, reinterpret_cast<double2 *>(out));
      ++h->launches;
      CU(cudaGetLastError());
      CU(cudaStreamSynchronize(h->stream));
      return TDDP4_OK;
    }
  }
  return fail(h, TDDP4_ERR_ARG, "unknown cache id %d", what);
}

int tddp4_layout(const tddp4 *h, int *n_sys, int *sys_mask, int *n_inst, int *inst_res, int *inst_sys, int *inst_sub) {
  if (!h) return TDDP4_ERR_ARG;
  const ModelTab &M = h->M;
  if (n_sys) *n_sys = M.n_sys;
  if (n_inst) *n_inst = M.n_inst;
  for (int i = 0; i < M.n_sys; ++i)
    if (sys_mask) sys_mask[i] = M.sys_mask[i];
  for (int j = 0; j < M.n_inst; ++j) {
    if (inst_res) inst_res[j] = M.inst[j].res;
    if (inst_sys) inst_sys[j] = M.inst[j].sys;
    if (inst_sub) inst_sub[j] = M.inst[j].sub;
  }
  return TDDP4_OK;
}

int tddp4_profile(tddp4 *h, int enable) {
  if (!h) return TDDP4_ERR_ARG;
  h->profiling = enable != 0;
  return TDDP4_OK;
}

int tddp4_profile_read(tddp4 *h, int kernel_id, double *total_ms, int64_t *launches, double *alg_bytes) {
  if (!h || kernel_id < 0 || kernel_id >= TDDP4_K_COUNT || !total_ms || !launches) return fail(h, TDDP4_ERR_ARG, "bad argument");
  drain_profile(h);
  *total_ms = h->prof_ms[kernel_id];
  *launches = h->prof_n[kernel_id];
  if (alg_bytes) *alg_bytes = h->prof_bytes[kernel_id];
  return TDDP4_OK;
}

int tddp4_profile_reset(tddp4 *h) {
  if (!h) return TDDP4_ERR_ARG;
  drain_profile(h);
  for (int i = 0; i < TDDP4_K_COUNT; ++i) { h->prof_ms[i] = 0; h->prof_n[i] = 0; h->prof_bytes[i] = 0; }
  return TDDP4_OK;
}

int64_t tddp4_launch_count(const tddp4 *h) { return h ? h->launches : 0; }

}  // extern "C"
