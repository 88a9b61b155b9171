// stream_kernels.cuh -- the per-call kernels of the NLL path that nvcc builds into the library:
//   nll_stream_kernel     steps 4+5+7   over cached coupling columns             (coupling / x / y / tau-only call)
//   nll_res_kernel, tres_kernel, prob_*  resolution mode (config 5) and per-event probabilities
// The two fused passes over the static caches are specialised to the model and compiled at run time:
//   colnll_jit.cuh        steps 2..5+7  over the static cache of the data set    (call after a mass or width moved)
//   gram_jit.cuh          steps 2+3+6   over the static cache of the normalisation set, fp64 tensor-core Gram
// All are HBM streams: every row is read exactly once per call with coalesced loads straight into registers (256-byte
// warp segments of 8-byte rows, 512-byte segments of the 16-byte columns), every load of an event requested before any
// arithmetic (9-36 loads in flight per thread), from STREAM_BLOCK-thread persistent blocks, two per SM.  Event i always
// belongs to thread (i mod stride) of the grid-stride decomposition, stride = gridDim.x * STREAM_BLOCK, and every thread
// visits its events in increasing order; nll_stream and colnll_jit are launched with the same grid and share their
// per-event arithmetic (nll_shared.cuh), so the fixed-order reduction returns bit-identical NLLs whether the columns were
// cached or rebuilt in the call.  Consecutive kernels overlap through programmatic dependent launch (jit_shared.cuh, pdl_*).
// (Measured on B200, 1M events x 136 B: a cp.async.bulk/mbarrier-staged version of the coupling-only pass with one block
// per SM ran at 35 us, this register-direct form at 26.7 us, a pure read of the same bytes at 22.6 us.)
#pragma once
#include "resolution.cuh"

namespace tddp4k {

// ------------------------------------------------------------------------------------------------
// Coupling-only call.  Reads K_c columns (16 B elements) and t: algorithmic traffic 16 K_c + 8 B per event.
// One event per thread per iteration (K_c + 1 independent loads in flight per thread, 72 registers at K_c = 8): the
// blocks of the NEXT kernel in the stream then fit next to this kernel's two blocks per SM, so consecutive calls
// overlap head to tail under programmatic dependent launch.  Measured on B200 (1 M events, K_c = 8, back to back):
// two events per iteration (128 registers, SM full) 21.3 us per call, this form 16.1 us; isolated both 22 us from
// first block start to result.  A reversed traversal on every other call (L2 reuse of the 136 MB stream in the 126 MB
// L2) gave 14.0 us but makes the per-thread product order depend on the call parity; not used.
template <int KC, bool SMALL>
__global__ void __launch_bounds__(STREAM_BLOCK, STREAM_BLOCKS_PER_SM)
nll_stream_kernel(const double2 *__restrict__ a, const double *__restrict__ t, int64_t ld, int64_t n,
                  const __grid_constant__ RateParams R, const double *__restrict__ G, double inv_n_norm, double sum_t,
                  double *__restrict__ partials, unsigned int *ticket, double *__restrict__ result, int early_wait, double seq,
                  unsigned long long *stamps /* in-kernel timing while profiling, else NULL */) {
  if (stamps && threadIdx.x == 0) atomicMin(stamps, global_ns());
  if (early_wait) pdl_wait();            // the predecessor wrote the columns
  pdl_launch_dependents();               // only after this kernel's own early wait: see the ordering note at pdl_wait()
  MantAcc la;
  const double yG = R.y * R.Gamma, xG = R.x * R.Gamma;
  const int64_t stride = (int64_t)gridDim.x * STREAM_BLOCK;
#pragma unroll 1
  for (int64_t i = (int64_t)blockIdx.x * STREAM_BLOCK + threadIdx.x; i < n; i += stride) {
    double2 v[KC];
#pragma unroll
    for (int c = 0; c < KC; ++c) v[c] = ldg_stream2(a + c * ld + i);
    double ti = ldg_stream1(t + i);
    double2 A = make_double2(0.0, 0.0), Ab = make_double2(0.0, 0.0);
#pragma unroll
    for (int c = 0; c < KC; ++c) amp_add(A, Ab, R.c[c][0], R.c[c][1], R.cbar[c][0], R.cbar[c][1], v[c]);
    la.add(bracket<SMALL>(A, Ab, yG * ti, xG * ti));
  }
  if (!early_wait) pdl_wait();
  nll_finish(R, KC, n, sum_t, la, G, inv_n_norm, partials, ticket, result, seq, stamps);
}

// P_i = e^{-Gamma t_i} B_i / N for parity and plots (tddp4_nll with prob_out): same per-event arithmetic as the
// NLL kernels, N read from the result slot the NLL kernel before it on the stream has written.
template <bool SMALL>
__global__ void __launch_bounds__(STREAM_BLOCK)
prob_kernel(const double2 *__restrict__ a, const double *__restrict__ t, int64_t ld, int64_t n, int KC,
            const __grid_constant__ RateParams R, const double *__restrict__ result, double *__restrict__ prob_out) {
  int64_t i = (int64_t)blockIdx.x * STREAM_BLOCK + threadIdx.x;
  if (i >= n) return;
  const double norm = result[2];
  double2 A = make_double2(0.0, 0.0), Ab = make_double2(0.0, 0.0);
  for (int c = 0; c < KC; ++c) amp_add(A, Ab, R.c[c][0], R.c[c][1], R.cbar[c][0], R.cbar[c][1], a[c * ld + i]);
  double ti = t[i];
  prob_out[i] = exp(-R.Gamma * ti) * bracket<SMALL>(A, Ab, R.y * R.Gamma * ti, R.x * R.Gamma * ti) / norm;
}

// Coupling-only call with per-event resolution (config 5): K_c columns + the eight time rows, 16 K_c + 64 B per event.
template <int KC>
__global__ void __launch_bounds__(STREAM_BLOCK, STREAM_BLOCKS_PER_SM)
nll_res_kernel(const double2 *__restrict__ a, const double *__restrict__ tr, int64_t ld, int64_t n,
               const __grid_constant__ RateParams R, const double *__restrict__ G, double inv_n_norm,
               double *__restrict__ partials, unsigned int *ticket, double *__restrict__ result, double seq) {
  __shared__ double s_S[4];
  MantAcc la;
  pdl_wait();                              // G is read first thing
  pdl_launch_dependents();
  block_phase_space_sums(R, G, KC, inv_n_norm, s_S);
  const int64_t stride = (int64_t)gridDim.x * STREAM_BLOCK;
#pragma unroll 1
  for (int64_t i = (int64_t)blockIdx.x * STREAM_BLOCK + threadIdx.x; i < n; i += stride) {
    double2 v[KC];
#pragma unroll
    for (int c = 0; c < KC; ++c) v[c] = ldg_stream2(a + c * ld + i);
    double2 A = make_double2(0.0, 0.0), Ab = make_double2(0.0, 0.0);
#pragma unroll
    for (int c = 0; c < KC; ++c) amp_add(A, Ab, R.c[c][0], R.c[c][1], R.cbar[c][0], R.cbar[c][1], v[c]);
    la.add(resolved_prob(A, Ab, tr + i, ld, s_S));
  }
  nll_finish<true>(R, KC, n, 0.0, la, G, inv_n_norm, partials, ticket, result, seq);
}
// P_i with resolution for prob_out
__global__ void __launch_bounds__(STREAM_BLOCK)
prob_res_kernel(const double2 *__restrict__ a, const double *__restrict__ tr, int64_t ld, int64_t n, int KC,
                const __grid_constant__ RateParams R, const double *__restrict__ G, double inv_n_norm,
                double *__restrict__ prob_out) {
  __shared__ double s_S[4];
  block_phase_space_sums(R, G, KC, inv_n_norm, s_S);
  int64_t i = (int64_t)blockIdx.x * STREAM_BLOCK + threadIdx.x;
  if (i >= n) return;
  double2 A = make_double2(0.0, 0.0), Ab = make_double2(0.0, 0.0);
  for (int c = 0; c < KC; ++c) amp_add(A, Ab, R.c[c][0], R.c[c][1], R.cbar[c][0], R.cbar[c][1], a[c * ld + i]);
  prob_out[i] = resolved_prob(A, Ab, tr + i, ld, s_S);
}

// The time rows of the data sample: psi[4], tint[4] per event (resolution.cuh).  Re-run when x, y, tau or the sample
// change; one thread per event; reads t and sigma_t (16 B), writes 64 B.  ALU-bound (3 exp, 6 erfcx, 3 Faddeeva).
constexpr int TRES_BLOCK = 128;
// parts: bit 0 = the real-lambda rows (psi_0, psi_2, T_0, T_2: they depend on y and tau), bit 1 = the complex-lambda rows
// (psi_1, psi_3, T_1, T_3: x and tau).  A step that moved only x (only y) rewrites only its half of the rows.
__global__ void __launch_bounds__(TRES_BLOCK)
tres_kernel(const __grid_constant__ FaddTab F, const double *__restrict__ t, const double *__restrict__ sigma_t, int64_t n,
            double x, double y, double Gamma, double t_lo, double t_hi, const TresTable *__restrict__ table,
            double *__restrict__ tr, int64_t ld, int parts) {
  __shared__ TresTable tab;
  for (int k = threadIdx.x; k < (int)(sizeof(TresTable) / sizeof(double)); k += TRES_BLOCK)
    reinterpret_cast<double *>(&tab)[k] = reinterpret_cast<const double *>(table)[k];
  __syncthreads();
  int64_t i = (int64_t)blockIdx.x * TRES_BLOCK + threadIdx.x;
  if (i >= n) return;
  const double ti = t[i], sig = sigma_t[i];
  const bool table_ok = tab.ok != 0;              // block-uniform
  double tint[4];
  if (table_ok) window_terms_table(tab, sig, tint);
  const double derf = table_ok ? 0.0 : erf_scaled(t_hi, sig) - erf_scaled(t_lo, sig);
  if (parts & 1) {
    const double lm = Gamma * (1.0 - y), lp = Gamma * (1.0 + y);
    const double hm = conv_exp_real(ti, lm, sig), hp = conv_exp_real(ti, lp, sig);
    tr[0 * ld + i] = 0.5 * (hm + hp);
    tr[2 * ld + i] = 0.5 * (hm - hp);
    if (!table_ok) {
      const double Im = window_real(t_lo, t_hi, lm, sig, derf), Ip = window_real(t_lo, t_hi, lp, sig, derf);
      tint[0] = 0.5 * (Im + Ip); tint[2] = 0.5 * (Im - Ip);
    }
    tr[4 * ld + i] = tint[0];
    tr[6 * ld + i] = tint[2];
  }
  if (parts & 2) {
    const double2 hx = conv_exp_complex(F, ti, Gamma, -Gamma * x, sig);
    tr[1 * ld + i] = hx.x;
    tr[3 * ld + i] = hx.y;
    if (!table_ok) {
      const double2 Ix = window_complex(F, t_lo, t_hi, Gamma, -Gamma * x, sig, derf);
      tint[1] = Ix.x; tint[3] = Ix.y;
    }
    tr[5 * ld + i] = tint[1];
    tr[7 * ld + i] = tint[3];
  }
}

// Time-integrated mode (use_resolution = 2): every event has the same eight "time quantities", the window integrals
// T_m themselves (psi_m = T_m: the rate integrated over the window; N_i = sum_m T_m S_m = N), so the resolution-mode
// kernels evaluate P_i = F(p_i) / N unchanged.  vals: the eight row constants.
struct Row8 { double v[8]; };
__global__ void __launch_bounds__(256) fill_rows_kernel(double *__restrict__ rows, int64_t ld, int64_t n, Row8 vals) {
  int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
  if (i >= n) return;
#pragma unroll
  for (int m = 0; m < 8; ++m) rows[m * ld + i] = vals.v[m];
}

// The derivative rows of the data sample for the gradient in resolution mode (resolution.cuh): 8 rows per event.
__global__ void __launch_bounds__(TRES_BLOCK)
tres_grad_kernel(const __grid_constant__ FaddTab F, const double *__restrict__ t, const double *__restrict__ sigma_t, int64_t n,
                 double x, double y, double Gamma, double t_lo, double t_hi, double *__restrict__ trg, int64_t ld) {
  int64_t i = (int64_t)blockIdx.x * TRES_BLOCK + threadIdx.x;
  if (i >= n) return;
  double d[8];
  time_term_derivatives(F, t[i], sigma_t[i], x, y, Gamma, t_lo, t_hi, d);
#pragma unroll
  for (int m = 0; m < 8; ++m) trg[m * ld + i] = d[m];
}

}  // namespace tddp4k
