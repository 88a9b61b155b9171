// stream_kernels.cuh -- the per-call kernels of the NLL path:
//   nll_stream_kernel     steps 4+5+7   over cached coupling columns             (coupling / x / y / tau-only call)
//   colnll_stream_kernel  steps 2..5+7  over the static cache of the data set    (call after a mass or width moved)
//   (gram_kernel.cuh:     steps 2+3+6   over the static cache of the normalisation set, fp64 tensor-core Gram)
//   nll_res_kernel, tres_kernel, prob_*  resolution mode (config 5) and per-event probabilities
// All are HBM streams: every row is read exactly once per call with coalesced loads straight into registers (256-byte
// warp segments of 8-byte rows, 512-byte segments of the 16-byte columns), every load of an event requested before any
// arithmetic (9-40 loads in flight per thread), from STREAM_BLOCK-thread persistent blocks, two per SM.  Event i always
// belongs to thread (i mod stride) of the grid-stride decomposition, stride = gridDim.x * STREAM_BLOCK, and every thread
// visits its events in increasing order; nll_stream and colnll_stream are launched with the same grid, so the fixed-order
// reduction returns bit-identical NLLs whether the columns were cached or rebuilt in the call.  Consecutive kernels
// overlap through programmatic dependent launch (pdl_* below).
// (Measured on B200, 1M events x 136 B: a cp.async.bulk/mbarrier-staged version of the coupling-only pass with one block
// per SM ran at 35 us, this register-direct form at 26.7 us, a pure read of the same bytes at 22.6 us.)
#pragma once
#include "resolution.cuh"

namespace tddp4k {

constexpr int STREAM_BLOCK = 256;
constexpr int STREAM_WARPS = STREAM_BLOCK / 32;
constexpr int STREAM_BLOCKS_PER_SM = 2;

// ------------------------------------------------------------------------------------------------
// sum_i log B_i without a log per event: B = m 2^e with m in [1,2); the mantissas are multiplied up and the
// exponents added as integers.  Partial results are merged by multiplication too (thread -> warp -> block -> grid,
// all in fixed order), so ONE log is taken per call:  sum log B = log(prod m) + ln2 * sum e.
struct MantAcc {
  double prod = 1.0;
  long long esum = 0;
  int bad = 0, since = 0;
  __device__ __forceinline__ void add(double B) {
    long long bits = __double_as_longlong(B);
    int e = (int)((bits >> 52) & 0x7ff);
    if (bits <= 0 || e == 0x7ff) { ++bad; return; }              // B <= 0 (sign bit or zero), inf, nan
    if (e == 0) {                                                 // subnormal: rescale first
      bits = __double_as_longlong(B * 0x1.0p64);
      e = (int)((bits >> 52) & 0x7ff) - 64;
    }
    esum += e - 1023;
    prod *= __longlong_as_double((bits & 0x000fffffffffffffLL) | 0x3ff0000000000000LL);
    if (++since == 512) renorm();
  }
  __device__ __forceinline__ void renorm() {
    long long bits = __double_as_longlong(prod);
    esum += (int)((bits >> 52) & 0x7ff) - 1023;
    prod = __longlong_as_double((bits & 0x000fffffffffffffLL) | 0x3ff0000000000000LL);
    since = 0;
  }
  // other must be renormalised (prod in [1,2))
  __device__ __forceinline__ void merge(double p, long long e, int b) { prod *= p; esum += e; bad += b; }
};
// butterfly over the warp: every lane ends with the warp's product (same bits in every lane)
__device__ __forceinline__ void warp_merge(MantAcc &m) {
  m.renorm();
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    double p = __shfl_xor_sync(0xffffffffu, m.prod, o);
    long long e = __shfl_xor_sync(0xffffffffu, m.esum, o);
    int b = __shfl_xor_sync(0xffffffffu, m.bad, o);
    m.merge(p, e, b);
  }
  m.renorm();
}

// one coupling column into the two amplitude sums of eq. (2); explicit FMAs: the same bits in every kernel
__device__ __forceinline__ void amp_add(double2 &A, double2 &Ab, double cr, double ci, double br, double bi, double2 v) {
  A.x = fma(cr, v.x, fma(-ci, v.y, A.x));
  A.y = fma(cr, v.y, fma(ci, v.x, A.y));
  Ab.x = fma(br, v.x, fma(-bi, v.y, Ab.x));
  Ab.y = fma(br, v.y, fma(bi, v.x, Ab.y));
}

// N from the Gram matrix in force (O-8, step 6): N = T1 (nAA + nBB) + T2 (nAA - nBB) - 2 T3 Re X - 2 T4 Im X,
// nAA = c^T G conj(c), nBB likewise for cbar, X = sum_kl c_k conj(cbar_l) G_kl.  One warp, (k,l) pairs strided over
// the lanes, fixed shuffle tree; every lane returns the same value.
__device__ __forceinline__ void gram_sums_warp(const RateParams &R, const double *__restrict__ G, int KC, double inv_n,
                                               double &nAA, double &nBB, double &xr, double &xi) {
  const int lane = threadIdx.x & 31;
  nAA = 0.0; nBB = 0.0; xr = 0.0; xi = 0.0;
  for (int q = lane; q < KC * KC; q += 32) {
    int k = q / KC, l = q % KC;
    double gr = __ldcg(G + q * 2) * inv_n, gi = __ldcg(G + q * 2 + 1) * inv_n;
    double ckr = R.c[k][0], cki = R.c[k][1], clr = R.c[l][0], cli = R.c[l][1];
    double bkr = R.cbar[k][0], bki = R.cbar[k][1], blr = R.cbar[l][0], bli = R.cbar[l][1];
    double pr = ckr * clr + cki * cli, pi = cki * clr - ckr * cli;
    nAA += pr * gr - pi * gi;
    pr = bkr * blr + bki * bli; pi = bki * blr - bkr * bli;
    nBB += pr * gr - pi * gi;
    pr = ckr * blr + cki * bli; pi = cki * blr - ckr * bli;
    xr += pr * gr - pi * gi;
    xi += pr * gi + pi * gr;
  }
  nAA = warp_sum(nAA); nBB = warp_sum(nBB); xr = warp_sum(xr); xi = warp_sum(xi);
}
__device__ __forceinline__ double norm_from_gram_warp(const RateParams &R, const double *__restrict__ G, int KC, double inv_n) {
  double nAA, nBB, xr, xi;
  gram_sums_warp(R, G, KC, inv_n, nAA, nBB, xr, xi);
  return R.T[0] * (nAA + nBB) + R.T[1] * (nAA - nBB) - 2.0 * R.T[2] * xr - 2.0 * R.T[3] * xi;
}

// Resolution mode (O-8, config 5): the phase-space sums S_1..S_4 = <w(|A|^2+|Abar|^2)>, <w(|A|^2-|Abar|^2)>, <w Re A Abar*>,
// <w Im A Abar*> must be known BEFORE the data pass, because the normalisation N_i = sum_m T_m(sigma_i) S_m is per
// event.  Warp 0 of every block derives them from the Gram matrix in force (same code, same bits in every block).
__device__ __forceinline__ void block_phase_space_sums(const RateParams &R, const double *__restrict__ G, int KC, double inv_n,
                                                       double *s_S /* shared [4] */) {
  if ((threadIdx.x >> 5) == 0) {
    double nAA, nBB, xr, xi;
    gram_sums_warp(R, G, KC, inv_n, nAA, nBB, xr, xi);
    if ((threadIdx.x & 31) == 0) { s_S[0] = nAA + nBB; s_S[1] = nAA - nBB; s_S[2] = xr; s_S[3] = xi; }
  }
  __syncthreads();
}
// P_i = R_i / N_i of one event from its amplitudes and its eight cached time quantities (rows psi[4], tint[4])
__device__ __forceinline__ double resolved_prob(double2 A, double2 Ab, const double *__restrict__ tr_i, int64_t ld,
                                                const double *s_S) {
  double v[8];
#pragma unroll
  for (int m = 0; m < 8; ++m) v[m] = ldg_stream1(tr_i + m * ld);
  double Rv = rate_form(bilinears(A, Ab), v[0], v[1], v[2], v[3]);
  double Nv = fma(s_S[0], v[4], fma(s_S[1], v[5], fma(-2.0 * s_S[2], v[6], __dmul_rn(-2.0 * s_S[3], v[7]))));
  return __ddiv_rn(Rv, Nv);
}

// common tail of the two NLL kernels (step 7, second pass).  Thread products -> warp -> block partial
// (prod, exponent sum, #bad); the last block to arrive merges the block partials in index order in warp 0 while
// warp 1 evaluates N, then thread 0 takes the one log and writes the result slot:
//   [0] sum log B, [1] sum t, [2] N, [3] NLL = Gamma sum t - sum log B + n log N, [4] #bad events,
//   [5] seq: the caller's sequence stamp, written LAST behind a system-wide fence -- when the slot lives in mapped host
//   memory the host polls this word instead of waiting on a CUDA event (see wait_slot() in tddp4_api.cu)
template <bool RES = false>
__device__ __forceinline__ void nll_finish(const RateParams &R, int KC, int64_t n, double sum_t, MantAcc la,
                                           const double *__restrict__ G, double inv_n, double *__restrict__ partials,
                                           unsigned int *ticket, double *__restrict__ result, double seq) {
  __shared__ double s_p[STREAM_WARPS];
  __shared__ long long s_e[STREAM_WARPS];
  __shared__ int s_b[STREAM_WARPS];
  __shared__ double s_norm;
  __shared__ bool last;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  warp_merge(la);
  if (lane == 0) { s_p[warp] = la.prod; s_e[warp] = la.esum; s_b[warp] = la.bad; }
  __syncthreads();
  if (threadIdx.x == 0) {
    MantAcc m;
#pragma unroll
    for (int w = 0; w < STREAM_WARPS; ++w) m.merge(s_p[w], s_e[w], s_b[w]);
    m.renorm();
    partials[3 * blockIdx.x] = m.prod;
    partials[3 * blockIdx.x + 1] = (double)m.esum;
    partials[3 * blockIdx.x + 2] = (double)m.bad;
    __threadfence();
    last = atomicAdd(ticket, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!last) return;
  __threadfence();
  // last block: every thread takes the block partials b = tid, tid + 256, ... (loads independent, issued together), warps
  // merge by butterfly, thread 0 merges the warps in order; warp 7 also evaluates N.  Fixed order: same bits every run.
  MantAcc m;
  {
    constexpr int PER = 8;                                // up to 8 * 256 = 2048 blocks
    double pp[PER], pe[PER], pb[PER];
#pragma unroll
    for (int r = 0; r < PER; ++r) {
      unsigned b = threadIdx.x + r * STREAM_BLOCK;
      bool ok = b < gridDim.x;
      pp[r] = ok ? __ldcg(partials + 3 * b) : 1.0;
      pe[r] = ok ? __ldcg(partials + 3 * b + 1) : 0.0;
      pb[r] = ok ? __ldcg(partials + 3 * b + 2) : 0.0;
    }
#pragma unroll
    for (int r = 0; r < PER; ++r) {
      m.merge(pp[r], (long long)pe[r], (int)pb[r]);
      m.renorm();
    }
    for (unsigned b = threadIdx.x + PER * STREAM_BLOCK; b < gridDim.x; b += STREAM_BLOCK) {   // larger grids: the slow way
      m.merge(__ldcg(partials + 3 * b), (long long)__ldcg(partials + 3 * b + 1), (int)__ldcg(partials + 3 * b + 2));
      m.renorm();
    }
  }
  warp_merge(m);
  __syncthreads();                                        // s_p .. s_b of the first stage are free
  if (lane == 0) { s_p[warp] = m.prod; s_e[warp] = m.esum; s_b[warp] = m.bad; }
  if (warp == STREAM_WARPS - 1) {
    double nv = norm_from_gram_warp(R, G, KC, inv_n);
    if (lane == 0) s_norm = nv;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    m = MantAcc();
#pragma unroll
    for (int w = 0; w < STREAM_WARPS; ++w) { m.merge(s_p[w], s_e[w], s_b[w]); m.renorm(); }
  }
  if (threadIdx.x == 0) {
    double norm = s_norm;
    double s0 = log(m.prod) + 0.693147180559945309417 * (double)m.esum;
    // -sum log(e^{-Gamma t} B / N) = Gamma sum t - sum log B + n log N
    double nll = R.Gamma * sum_t - s0 + (double)n * log(norm);
    if (RES) { nll = -s0; sum_t = 0.0; }                 // the accumulated values were P_i = R_i / N_i already
    if (m.bad > 0 || !(norm > 0.0)) nll = INFINITY;
    result[0] = s0; result[1] = sum_t; result[2] = norm; result[3] = nll; result[4] = (double)m.bad;
    *ticket = 0;
    if (seq != 0.0) {                       // 0: nobody polls this slot (batched / device-side results)
      __threadfence_system();
      *reinterpret_cast<volatile double *>(result + 5) = seq;
    }
  }
}

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
                  double *__restrict__ partials, unsigned int *ticket, double *__restrict__ result, int early_wait, double seq) {
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
  nll_finish(R, KC, n, sum_t, la, G, inv_n_norm, partials, ticket, result, seq);
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

// ------------------------------------------------------------------------------------------------
// steps 2+3 of ONE event from the tile-major static cache (tables.h).  ev = address of (row 0, this event): every row is
// ev[row * 32], so with the loops unrolled to the table maxima (one warp-uniform guard per load batch) every load carries an
// immediate offset and every table entry / lineshape constant is an immediate-indexed constant-bank operand.
// Lineshapes: T_R of every de-duplicated instance goes to the thread's own slots sTl[slot * 32] of its warp's
// scratch (chains index it through the model tables, so it cannot live in registers); slot n_inst4 holds the unit
// lineshape 1 + 0i that non-resonant and padded terms multiply by.  Loads are issued in batches of GI instances and GT
// terms, the first f batch BEFORE the lineshape arithmetic: 2 GI + GT loads in flight per thread (40 for config 3).
// These kernels are bound by memory-level parallelism, not by bytes or issue slots: with batches of 4 instances the
// Gram kernel ran at 0.51 of the HBM roofline, with (12, 16) at 0.71.  (Measured and rejected: software-pipelining the
// next tile's loads behind this tile's arithmetic, 312 us against 240 us; register-resident one-batch forms without the
// group guards, which ptxas schedules into spills.)
template <int GI>
__device__ __forceinline__ void lineshapes_to_scratch(const StreamTab &S, const LineParams &LP, const double *__restrict__ ev,
                                                      double2 *sTl) {
  const double *g_ev = ev + S.g_off;
#pragma unroll
  for (int j0 = 0; j0 < MAX_INST; j0 += GI) {
    if (j0 < S.n_inst4) {
      double sv[GI], gv[GI];
#pragma unroll
      for (int u = 0; u < GI; ++u) {
        sv[u] = __ldg(ev + S.inst_soff[j0 + u]);
        gv[u] = ldg_stream1(g_ev + (j0 + u) * 32);
      }
#pragma unroll
      for (int u = 0; u < GI; ++u) sTl[(j0 + u) * 32] = breit_wigner(LP.m0sq[j0 + u], LP.gam[j0 + u], sv[u], gv[u]);
    }
  }
}
// The f rows of the first term group, issued BEFORE the lineshape arithmetic so that they are in flight with it.
template <int GT>
__device__ __forceinline__ void prefetch_f(const StreamTab &S, const double *__restrict__ ev, double (&fv)[GT]) {
  const double *f_ev = ev + S.f_off;
#pragma unroll
  for (int u = 0; u < GT; ++u) fv[u] = ldg_stream1(f_ev + u * 32);
}
// Component products summed into coupling columns: a_kappa = sum_{k in kappa} f_k T_{R1(k)} T_{R2(k)} (terms are sorted
// by coupling).  flush(kappa, a_kappa) is called once per non-empty column, in order.  fv: first group, preloaded.
template <int GT, class Flush>
__device__ __forceinline__ void columns_from_scratch(const StreamTab &S, const double *__restrict__ ev, const double2 *sTl,
                                                     double (&fv)[GT], Flush &&flush) {
  const double *f_ev = ev + S.f_off;
  double2 acc = make_double2(0.0, 0.0);
#pragma unroll
  for (int k0 = 0; k0 < MAX_TERMS; k0 += GT) {
    if (k0 < S.n_terms4) {
      if (k0 > 0) {
#pragma unroll
        for (int u = 0; u < GT; ++u) fv[u] = ldg_stream1(f_ev + (k0 + u) * 32);
      }
      // Two phases per sub-batch of TB terms: first every lineshape product (shared-memory reads only), then the sums and
      // the flushes.  A flush stores to shared memory (the Gram kernel's X tile) at a run-time address, which the compiler
      // must assume to alias the lineshape slots: with one loop it kept every term's two LDS behind the previous term's
      // store, sixteen serial LDS -> DMUL -> DFMA chains per event (34 % of the Gram kernel's warp samples).
      constexpr int TB = GT < 8 ? GT : 8;
#pragma unroll
      for (int u0 = 0; u0 < GT; u0 += TB) {
        double2 TT[TB];
#pragma unroll
        for (int u = 0; u < TB; ++u) TT[u] = cmul(sTl[S.term_t0[k0 + u0 + u]], sTl[S.term_t1[k0 + u0 + u]]);
#pragma unroll
        for (int u = 0; u < TB; ++u) {
          const int k = k0 + u0 + u;
          acc.x = fma(fv[u0 + u], TT[u].x, acc.x);
          acc.y = fma(fv[u0 + u], TT[u].y, acc.y);
          if (S.term_last[k]) {
            flush((int)S.term_col[k], acc);
            acc = make_double2(0.0, 0.0);
          }
        }
      }
    }
  }
}
__host__ __device__ inline size_t lineshape_scratch_bytes(int n_inst4) { return (size_t)(n_inst4 + 1) * 32 * sizeof(double2); }
// ------------------------------------------------------------------------------------------------
// Call after a mass or width moved, data set.  Reads the s rows in use, the g rows, the f rows and t; writes every
// coupling column back (for the coupling-only calls that follow) and finishes the NLL in the same pass.
inline size_t colnll_smem_bytes(int n_inst4) { return STREAM_WARPS * lineshape_scratch_bytes(n_inst4); }

// GI, GT: load-batch sizes (instances, terms) of the model's size class; the tables are padded to multiples of them.
template <bool SMALL, bool RES, int GI, int GT>
__global__ void __launch_bounds__(STREAM_BLOCK, STREAM_BLOCKS_PER_SM)
colnll_stream_kernel(const __grid_constant__ StreamTab S, const __grid_constant__ LineParams LP,
                     const double *__restrict__ cache, const double *__restrict__ t, int64_t ld, int64_t n,
                     double2 *__restrict__ a,
                     const __grid_constant__ RateParams R, const double *__restrict__ G, double inv_n_norm, double sum_t,
                     double *__restrict__ partials, unsigned int *ticket, double *__restrict__ result, int early_wait,
                     uint32_t store_mask /* bit kappa: the stored column kappa is stale and is rewritten */, double seq) {
  extern __shared__ __align__(16) char smem_raw[];
  __shared__ double s_S[4];
  if (RES || early_wait) pdl_wait();       // the predecessor reads the columns this kernel rewrites (or RES: G first)
  pdl_launch_dependents();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  double2 *sTl = reinterpret_cast<double2 *>(smem_raw + (size_t)warp * lineshape_scratch_bytes(S.n_inst4)) + lane;
  sTl[S.n_inst4 * 32] = make_double2(1.0, 0.0);        // unit lineshape slot
  MantAcc la;
  const double yG = R.y * R.Gamma, xG = R.x * R.Gamma;
  const int64_t stride = (int64_t)gridDim.x * STREAM_BLOCK;
  if (RES) block_phase_space_sums(R, G, S.n_kc, inv_n_norm, s_S);
  int64_t i = (int64_t)blockIdx.x * STREAM_BLOCK + threadIdx.x;
#pragma unroll
  for (int d = 1; d < PF_DIST; ++d)
    if (lane == 0 && i + d * stride < n) prefetch_l2_bulk(tile_event(cache, S.R, i + d * stride) + S.skip, (uint32_t)(S.R * 32 - S.skip) * 8u);
#pragma unroll 1
  for (; i < n; i += stride) {
    if (PF_DIST > 0 && lane == 0 && i + PF_DIST * stride < n) prefetch_l2_bulk(tile_event(cache, S.R, i + PF_DIST * stride) + S.skip, (uint32_t)(S.R * 32 - S.skip) * 8u);
    double ti = RES ? 0.0 : ldg_stream1(t + i);            // RES: t points at the time rows [8][ld]
    const double *ev = tile_event(cache, S.R, i);
    double fv[GT];
    prefetch_f<GT>(S, ev, fv);
    lineshapes_to_scratch<GI>(S, LP, ev, sTl);
    double2 A = make_double2(0.0, 0.0), Ab = make_double2(0.0, 0.0);
    columns_from_scratch<GT>(S, ev, sTl, fv, [&](int kap, double2 col) {
      // a column none of whose lineshapes moved is recomputed to the bits already stored: skip its 16-byte store
      if ((store_mask >> kap) & 1u) a[(int64_t)kap * ld + i] = col;
      amp_add(A, Ab, R.c[kap][0], R.c[kap][1], R.cbar[kap][0], R.cbar[kap][1], col);
    });
    if (RES) la.add(resolved_prob(A, Ab, t + i, ld, s_S));
    else la.add(bracket<SMALL>(A, Ab, yG * ti, xG * ti));
  }
  if (!(RES || early_wait)) pdl_wait();
  nll_finish<RES>(R, S.n_kc, n, sum_t, la, G, inv_n_norm, partials, ticket, result, seq);
}

}  // namespace tddp4k
