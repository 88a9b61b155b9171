// stream_kernels.cuh -- the per-call kernels of the NLL path:
//   nll_stream_kernel     steps 4+5+7   over cached coupling columns             (coupling / x / y / tau-only call)
//   colnll_stream_kernel  steps 2..5+7  over the static cache of the data set    (call after a mass or width moved)
//   gram_stream_kernel    steps 2+3+6   over the static cache of the normalisation set (fp64 tensor-core Gram)
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

__host__ __device__ constexpr size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// read-once loads: no L1 allocation
__device__ __forceinline__ double2 ldg_stream2(const double2 *p) {
  double2 v;
  asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
  return v;
}
__device__ __forceinline__ double ldg_stream1(const double *p) {
  double v;
  asm volatile("ld.global.nc.L1::no_allocate.f64 %0, [%1];" : "=d"(v) : "l"(p));
  return v;
}

// Programmatic dependent launch (the host launches the per-call kernels with programmatic stream serialization): a kernel
// lets its successor's blocks become resident as soon as its own blocks exit, so the successor's launch latency, ramp-up
// and read-only streaming overlap this kernel's tail and final reduction.  pdl_wait() blocks until the predecessor grid
// has completed and its memory is visible; it sits in front of the first access to anything the predecessor may read or
// write (partials, ticket, G, result slots; the columns when the predecessor or this kernel writes them).
// Ordering rule: a successor may become resident as soon as every block of this kernel has executed
// launch_dependents -- possibly while this kernel's own predecessor is still running.  A successor that skips its early
// wait must therefore never conflict with that older kernel: (i) a kernel that has an early wait triggers only after it,
// (ii) the Gram kernel, after which the column-writing kernel skips its early wait, triggers only after its late wait,
// (iii) an NLL kernel without early wait may trigger at once: whatever follows it either waits early or only reads what
// no kernel before it writes.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// One lane asks the memory system to bring a whole contiguous region into L2 (no destination, no register, no scoreboard):
// the tile-major cache makes the NEXT tile of a warp one such region, so its loads later hit L2 instead of HBM.
__device__ __forceinline__ void prefetch_l2_bulk(const void *p, uint32_t bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}

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
#pragma unroll
      for (int u = 0; u < GT; ++u) {
        const int k = k0 + u;
        double2 T = cmul(sTl[S.term_t0[k]], sTl[S.term_t1[k]]);
        acc.x = fma(fv[u], T.x, acc.x);
        acc.y = fma(fv[u], T.y, acc.y);
        if (S.term_last[k]) {
          flush((int)S.term_col[k], acc);
          acc = make_double2(0.0, 0.0);
        }
      }
    }
  }
}
__host__ __device__ inline size_t lineshape_scratch_bytes(int n_inst4) { return (size_t)(n_inst4 + 1) * 32 * sizeof(double2); }
// address of (row 0, event i) in a tile-major cache of R rows
__device__ __forceinline__ const double *tile_event(const double *__restrict__ cache, int R, int64_t i) {
  return cache + ((i >> 5) * R) * 32 + (i & 31);
}

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
#pragma unroll 1
  for (; i < n; i += stride) {
    if (lane == 0 && i + stride < n) prefetch_l2_bulk(tile_event(cache, S.R, i + stride) + S.skip, (uint32_t)(S.R * 32 - S.skip) * 8u);
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

// ------------------------------------------------------------------------------------------------
// step 6: Hermitian Gram matrix G_kl = sum_j w_j a_k(p_j) conj(a_l(p_j)) over the normalisation sample, fused with
// steps 2+3: the columns of the normalisation sample are never stored.  With x_j = (Re a_0, Im a_0, Re a_1, ...)
// the real matrix X^T diag(w) X holds every Re/Im piece of G, and it is a dense contraction over events: it runs on
// the fp64 tensor cores (mma.sync m8n8k4, SASS DMMA), the only place of the path where they apply (north_star).
//   G_kl.re = XtX[2k][2l] + XtX[2k+1][2l+1],   G_kl.im = XtX[2k+1][2l] - XtX[2k][2l+1].
// One thread per event computes the columns into its row of the warp's X tile (padded, conflict-free fragments);
// the warp then feeds its 32 events, 4 at a time, through the MMA.  NB = number of 8-feature blocks.
// Reads the s rows in use, the g rows, the f rows, and w if the sample is weighted.
// Deterministic: per-warp accumulation in event order, warps then blocks summed in index order.
// X tile of a warp: row = event, gram_stride(NB) = 8 NB + 2 doubles per row (F = 8 NB features, the weight at [F]).
// Both access patterns are bank-conflict free: a lane's 16-byte column stores land in slot (e (4 NB + 1) + kappa) mod 8,
// distinct over the 8 lanes of a wavefront; MMA group g takes the four events e = 8 (g >> 1) + 2 (lane & 3) + (g & 1), so
// the fragment loads of a half-warp hit the 8-byte banks (phi + 4 (lane & 3) + const) mod 16, phi = lane >> 2.
// (Measured: rows of 20 doubles with groups of consecutive events had 2-way store conflicts, 7.2 M conflict
// wavefronts per 4 M events with the LSU data pipe 83 % busy; this layout: Gram kernel 215 -> 211 us.)
__host__ __device__ constexpr int gram_stride(int NB) { return 8 * NB + 2; }
constexpr int GRAM_GROUP = 16;        // blocks per group of the two-level grid reduction
constexpr int MAX_TICKETS = 1 + 256;  // grid ticket + group tickets (grids up to 4096 blocks)
inline size_t gram_warp_scratch(int NB, int n_inst4) {
  return align_up(lineshape_scratch_bytes(n_inst4), 128) + align_up((size_t)32 * gram_stride(NB) * sizeof(double), 128);
}
inline size_t gram_smem_bytes(int NB, int n_inst4) {
  size_t work = STREAM_WARPS * gram_warp_scratch(NB, n_inst4), red = (size_t)STREAM_WARPS * NB * NB * 64 * sizeof(double);
  return work > red ? work : red;
}

__device__ __forceinline__ void dmma884(double &c0, double &c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

template <int NB, int GI, int GT>
__global__ void __launch_bounds__(STREAM_BLOCK, STREAM_BLOCKS_PER_SM)
gram_stream_kernel(const __grid_constant__ StreamTab S, const __grid_constant__ LineParams LP,
                   const double *__restrict__ cache, int64_t n,
                   double *__restrict__ partials /* [grid][64 NB NB] */, unsigned int *ticket,
                   double *__restrict__ G /* [KC][KC][2] sums, Hermitian, full */) {
  constexpr int F = 8 * NB, STRIDE = gram_stride(NB), NP = NB * (NB + 1) / 2, WARPS = STREAM_WARPS;
  extern __shared__ __align__(16) char smem_raw[];
  __shared__ bool last;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int KC = S.n_kc;
  const size_t t_bytes = align_up(lineshape_scratch_bytes(S.n_inst4), 128);
  const size_t x_bytes = align_up((size_t)32 * STRIDE * sizeof(double), 128);
  char *scratch = smem_raw + (size_t)warp * (t_bytes + x_bytes);
  double2 *sTl = reinterpret_cast<double2 *>(scratch) + lane;  // [n_inst][32], this lane's slots
  double *Xs = reinterpret_cast<double *>(scratch + t_bytes);  // [32][STRIDE]: row = event, F features + weight
  double *row = Xs + lane * STRIDE;
  sTl[S.n_inst4 * 32] = make_double2(1.0, 0.0);                // unit lineshape slot
#pragma unroll
  for (int c = 0; c < STRIDE; ++c) row[c] = 0.0;                // features beyond 2 K_c stay zero
  double acc[NP][2];
#pragma unroll
  for (int q = 0; q < NP; ++q) acc[q][0] = acc[q][1] = 0.0;
  const int64_t stride = (int64_t)gridDim.x * STREAM_BLOCK;
  // whole warps iterate together (the MMA is warp-wide).  The cache is allocated and zero-filled in whole tiles, so the
  // lanes of a ragged last tile compute on zeros: f = 0 gives zero columns, and their weight is forced to 0.
  auto mma_tile = [&]() {
    __syncwarp();
    const double *base = Xs + (2 * (lane & 3)) * STRIDE + (lane >> 2);
#pragma unroll
    for (int grp = 0; grp < 8; ++grp) {                  // 4 events per MMA, 8 groups per warp tile
      const double *r = base + (8 * (grp >> 1) + (grp & 1)) * STRIDE;
      double wv = r[F - (lane >> 2)];
      double x[NB];
#pragma unroll
      for (int b = 0; b < NB; ++b) x[b] = r[8 * b];
      int q = 0;
#pragma unroll
      for (int bi = 0; bi < NB; ++bi) {
        double aw = wv * x[bi];
#pragma unroll
        for (int bj = bi; bj < NB; ++bj, ++q) dmma884(acc[q][0], acc[q][1], aw, x[bj]);
      }
    }
    __syncwarp();                                        // the X tile is free again
  };
  int64_t i0 = (int64_t)blockIdx.x * STREAM_BLOCK + warp * 32;
#pragma unroll 1
  for (; i0 < n; i0 += stride) {
    if (lane == 0 && i0 + stride < n) prefetch_l2_bulk(tile_event(cache, S.R, i0 + stride) + S.skip, (uint32_t)(S.R * 32 - S.skip) * 8u);
    const double *ev = tile_event(cache, S.R, i0 + lane);
    double wj = S.w_off >= 0 ? ldg_stream1(ev + S.w_off) : 1.0;
    double fv[GT];
    prefetch_f<GT>(S, ev, fv);
    lineshapes_to_scratch<GI>(S, LP, ev, sTl);
    columns_from_scratch<GT>(S, ev, sTl, fv, [&](int kap, double2 col) { *reinterpret_cast<double2 *>(row + 2 * kap) = col; });
    row[F] = i0 + lane < n ? wj : 0.0;
    mma_tile();
  }
  __syncthreads();                                       // all scratch is free
  // block reduction in warp order, block partial = upper 8x8 blocks of X^T W X
  double *Ws = reinterpret_cast<double *>(smem_raw);     // [WARPS][NB*NB][64]
  {
    int q = 0;
#pragma unroll
    for (int bi = 0; bi < NB; ++bi)
#pragma unroll
      for (int bj = bi; bj < NB; ++bj, ++q) {
        double *dst = Ws + ((warp * NB + bi) * NB + bj) * 64;
        dst[(lane >> 2) * 8 + 2 * (lane & 3)] = acc[q][0];      // C fragment: row lane/4, cols 2 (lane%4) + {0,1}
        dst[(lane >> 2) * 8 + 2 * (lane & 3) + 1] = acc[q][1];
      }
  }
  __syncthreads();
  pdl_wait();                              // partials, ticket and G may still be in use by the predecessor
  pdl_launch_dependents();                 // not earlier: a successor that skips its early wait relies on this kernel's
                                           // predecessors being complete once it becomes resident
  for (int e = tid; e < NB * NB * 64; e += STREAM_BLOCK) {
    int bi = e / (NB * 64), bj = (e / 64) % NB;
    if (bi > bj) continue;
    double sum = 0.0;
#pragma unroll
    for (int wp = 0; wp < WARPS; ++wp) sum += Ws[wp * NB * NB * 64 + e];
    partials[(int64_t)blockIdx.x * NB * NB * 64 + e] = sum;
  }
  // Two-level, fixed-order reduction over the grid.  Blocks form groups of GRAM_GROUP consecutive blocks; the last block
  // of a group to arrive (group ticket) adds the group's partials in block order, the last group to finish (grid ticket)
  // adds the group sums in group order.  Every level is one round of independent loads: two L2 round trips after the
  // last block partial instead of one block pulling all gridDim.x partials (455 KB at K_c = 8) through a single SM.
  const unsigned n_groups = (gridDim.x + GRAM_GROUP - 1) / GRAM_GROUP, grp = blockIdx.x / GRAM_GROUP;
  const unsigned g_first = grp * GRAM_GROUP, g_size = min((unsigned)GRAM_GROUP, gridDim.x - g_first);
  __threadfence();
  __syncthreads();
  if (tid == 0) last = atomicAdd(ticket + 1 + grp, 1u) == g_size - 1;
  __syncthreads();
  if (!last) return;
  __threadfence();
  double *gsum = partials + (int64_t)gridDim.x * NB * NB * 64;        // [n_groups][NB*NB*64]
  for (int e = tid; e < NB * NB * 64; e += STREAM_BLOCK) {
    int bi = e / (NB * 64), bj = (e / 64) % NB;
    if (bi > bj) continue;
    double v[GRAM_GROUP];
#pragma unroll
    for (int c = 0; c < GRAM_GROUP; ++c) v[c] = (unsigned)c < g_size ? __ldcg(partials + (int64_t)(g_first + c) * NB * NB * 64 + e) : 0.0;
    double sum = 0.0;
#pragma unroll
    for (int c = 0; c < GRAM_GROUP; ++c) sum += v[c];
    gsum[(int64_t)grp * NB * NB * 64 + e] = sum;
  }
  __threadfence();
  __syncthreads();
  if (tid == 0) { ticket[1 + grp] = 0; last = atomicAdd(ticket, 1u) == n_groups - 1; }
  __syncthreads();
  if (!last) return;
  __threadfence();
  double *XtX = Ws;                                      // [NB][NB][64], reused
  for (int e = tid; e < NB * NB * 64; e += STREAM_BLOCK) {
    int bi = e / (NB * 64), bj = (e / 64) % NB;
    if (bi > bj) continue;
    double sum = 0.0;
    unsigned g = 0;
    for (; g + 8 <= n_groups; g += 8) {
      double v[8];
#pragma unroll
      for (int c = 0; c < 8; ++c) v[c] = __ldcg(gsum + (int64_t)(g + c) * NB * NB * 64 + e);
#pragma unroll
      for (int c = 0; c < 8; ++c) sum += v[c];
    }
    for (; g < n_groups; ++g) sum += __ldcg(gsum + (int64_t)g * NB * NB * 64 + e);
    XtX[e] = sum;
  }
  __syncthreads();
  auto xtx = [&](int m, int nn) {                        // symmetric: only the upper triangle is ever read
    if (m > nn) { int tmp = m; m = nn; nn = tmp; }
    return XtX[((m >> 3) * NB + (nn >> 3)) * 64 + (m & 7) * 8 + (nn & 7)];
  };
  for (int q = tid; q < KC * KC; q += STREAM_BLOCK) {
    int kk = q / KC, l = q % KC;
    double re = xtx(2 * kk, 2 * l) + xtx(2 * kk + 1, 2 * l + 1);
    double im = xtx(2 * kk + 1, 2 * l) - xtx(2 * kk, 2 * l + 1);
    if (kk == l) im = 0.0;
    G[q * 2] = re;
    G[q * 2 + 1] = im;
  }
  if (tid == 0) *ticket = 0;
}

}  // namespace tddp4k
