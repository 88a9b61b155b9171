// nll_shared.cuh -- the per-event arithmetic of eq. (1) and the deterministic -sum log reduction
// (SURVEY.md 8(a) rows 4, 5, 7), shared by the kernels nvcc builds into libtddp4.so (stream_kernels.cuh, grad_kernels.cuh)
// and by the model-specialised data pass the library compiles at run time (colnll_jit.cuh).  No system header (NVRTC has
// none).  Every sum of products is written with explicit fma / __dmul_rn, so the same event gives the same bits in every
// kernel and under either compiler front end: cached and rebuilt calls return bit-identical NLLs.
#pragma once
#include "jit_shared.cuh"

namespace tddp4k {

#ifndef TDDP4_MAX_KC
#define TDDP4_MAX_KC 16            // = MAX_KC of tables.h (static_assert there)
#endif
struct RateParams {                // eq. (1) and O-8
  double c[TDDP4_MAX_KC][2];
  double cbar[TDDP4_MAX_KC][2];
  double x, y, Gamma;
  double T[4];                     // time integrals of cosh, cos, sinh, sin terms over the window
  double t_lo, t_hi;
  int use_resolution;
};


constexpr int STREAM_BLOCK = 256;
constexpr int STREAM_WARPS = STREAM_BLOCK / 32;
constexpr int STREAM_BLOCKS_PER_SM = 2;


__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// eq. (1): bracket B from A, Abar and the mixing phases u = y Gamma t, v = x Gamma t.
// SMALL (|u|, |v| < 1/4, guaranteed by the host): cosh, sinh, cos, sin as Taylor polynomials up to u^12 / u^13;
// the first omitted term is below 4e-20 of the leading one.
// the four time functions of eq. (1) at mixing phases u = y Gamma t, v = x Gamma t
template <bool SMALL>
__device__ __forceinline__ void mixing_functions(double u, double v, double &ch, double &sh, double &cs, double &sn) {
  if (SMALL) {
    const double c2 = 1.0 / 2, c4 = 1.0 / 24, c6 = 1.0 / 720, c8 = 1.0 / 40320, c10 = 1.0 / 3628800, c12 = 1.0 / 479001600;
    const double s3 = 1.0 / 6, s5 = 1.0 / 120, s7 = 1.0 / 5040, s9 = 1.0 / 362880, s11 = 1.0 / 39916800, s13 = 1.0 / 6227020800.0;
    double u2 = u * u, v2 = v * v;
    ch = fma(u2, fma(u2, fma(u2, fma(u2, fma(u2, fma(u2, c12, c10), c8), c6), c4), c2), 1.0);
    sh = u * fma(u2, fma(u2, fma(u2, fma(u2, fma(u2, fma(u2, s13, s11), s9), s7), s5), s3), 1.0);
    cs = fma(v2, fma(v2, fma(v2, fma(v2, fma(v2, fma(v2, c12, -c10), c8), -c6), c4), -c2), 1.0);
    sn = v * fma(v2, fma(v2, fma(v2, fma(v2, fma(v2, fma(v2, s13, -s11), s9), -s7), s5), -s3), 1.0);
  } else {
    double e = exp(u), ei = 1.0 / e;
    ch = 0.5 * (e + ei);
    sh = 0.5 * (e - ei);
    sincos(v, &sn, &cs);
  }
}
// |A|^2, |Abar|^2, Re(A conj(Abar)), Im(A conj(Abar)) and the bracket itself with every contraction written out
// (fma / __dmul_rn): the NLL, column-rebuilding and gradient kernels must produce the same bits for the same event, and
// nvcc's default -fmad=true would otherwise be free to contract the sums differently per template instantiation.
struct Bilinears { double aa, bb, cre, cim; };
__device__ __forceinline__ Bilinears bilinears(double2 A, double2 Ab) {
  Bilinears q;
  q.aa = fma(A.x, A.x, __dmul_rn(A.y, A.y));
  q.bb = fma(Ab.x, Ab.x, __dmul_rn(Ab.y, Ab.y));
  q.cre = fma(A.x, Ab.x, __dmul_rn(A.y, Ab.y));
  q.cim = fma(A.y, Ab.x, -__dmul_rn(A.x, Ab.y));
  return q;
}
// (aa + bb) f0 + (aa - bb) f1 - 2 cre f2 - 2 cim f3: eq. (1) with f = (cosh, cos, sinh, sin), or its convolved / integrated forms
__device__ __forceinline__ double rate_form(const Bilinears &q, double f0, double f1, double f2, double f3) {
  return fma(__dadd_rn(q.aa, q.bb), f0, fma(__dsub_rn(q.aa, q.bb), f1, fma(-2.0 * q.cre, f2, __dmul_rn(-2.0 * q.cim, f3))));
}
template <bool SMALL>
__device__ __forceinline__ double bracket(double2 A, double2 Ab, double u, double v) {
  double ch, sh, sn, cs;
  mixing_functions<SMALL>(u, v, ch, sh, cs, sn);
  return rate_form(bilinears(A, Ab), ch, cs, sh, sn);
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
__device__ __forceinline__ double resolved_prob(double2 A, double2 Ab, const double *__restrict__ tr_i, long long ld,
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
// %globaltimer: nanoseconds on one clock for the whole GPU (in-kernel timing of tddp4_profile, below)
__device__ __forceinline__ unsigned long long global_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}
// stamps (profiling only, else NULL): [0] earliest block start of this launch (atomicMin by the kernel's blocks), [1] sum
// over launches of (result written - earliest start) in ns, [2] launches counted.
template <bool RES = false>
__device__ __forceinline__ void nll_finish(const RateParams &R, int KC, long long n, double sum_t, MantAcc la,
                                           const double *__restrict__ G, double inv_n, double *__restrict__ partials,
                                           unsigned int *ticket, double *__restrict__ result, double seq,
                                           unsigned long long *stamps = nullptr) {
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
    if (m.bad > 0 || !(norm > 0.0)) nll = __longlong_as_double(0x7ff0000000000000LL);   // +inf (no math.h under NVRTC)
    result[0] = s0; result[1] = sum_t; result[2] = norm; result[3] = nll; result[4] = (double)m.bad;
    *ticket = 0;
    if (seq != 0.0) {                       // 0: nobody polls this slot (batched / device-side results)
      __threadfence_system();
      *reinterpret_cast<volatile double *>(result + 5) = seq;
    }
    if (stamps) {
      const unsigned long long t1 = global_ns(), t0 = *reinterpret_cast<volatile unsigned long long *>(stamps);
      atomicAdd(stamps + 1, t1 - t0);
      atomicAdd(stamps + 2, 1ull);
      *reinterpret_cast<volatile unsigned long long *>(stamps) = ~0ull;
    }
  }
}

}  // namespace tddp4k
