// resolution.cuh -- per-event Gaussian decay-time resolution (O-8, BASELINE config 5), sm_100a, fp64.
// Every e^{-lambda t} of eq. (1) becomes its convolution with a Gaussian of width sigma,
//   h(t; lambda, sigma) = 1/2 exp(lambda^2 sigma^2/2 - lambda t) erfc(u),   u = (lambda sigma^2 - t) / (sqrt2 sigma),
// lambda = Gamma(1 -+ y) (real) for the cosh/sinh terms and Gamma(1 - i x) (complex) for the cos/sin terms; the
// normalisation integrates h over the decay-time window with the antiderivative
//   H(t) = [erf(t / (sqrt2 sigma)) - 2 h(t)] / (2 lambda).
// Evaluation (no overflow, no cancellation): with g0 = exp(-t^2 / (2 sigma^2)) and the Faddeeva function w,
//   Re u >= 0:  h = 1/2 g0 w(i u);      Re u < 0:  h = exp(lambda^2 sigma^2/2 - lambda t) - 1/2 g0 w(-i u),
// so w is only ever needed in the closed upper half plane.  Real lambda: w(i u) = erfcx(u) (CUDA intrinsic).
// Complex lambda: Weideman's rational expansion of w (J.A.C. Weideman, SIAM J. Numer. Anal. 31 (1994) 1497),
//   w(z) ~ 2 p(Z) / (L - i z)^2 + (1/sqrt(pi)) / (L - i z),  Z = (L + i z)/(L - i z),  p = sum_{n<N} a_{n+1} Z^n,
// N = 40, L = sqrt(N / sqrt2); the a_n are the cosine coefficients of exp(-t^2)(L^2 + t^2) under t = L tan(theta/2),
// computed on the host at tddp4_create (fadd_coefficients below).  Measured against scipy.special.wofz on
// Im z in [0, 9], |Re z| < 1.5: relative error < 6e-15.
#pragma once
#include <math.h>

namespace tddp4k {

constexpr int FADD_N = 40;
struct FaddTab {
  double L;
  double a[FADD_N];   // a[0] multiplies Z^(N-1) (Horner order)
};

// host: a_n = (1/(4N)) sum_{k=-2N+1}^{2N-1} f(t_k) cos(n theta_k), theta_k = k pi/(2N), t_k = L tan(theta_k/2)
inline void fadd_coefficients(FaddTab &F) {
  const int N = FADD_N, M = 2 * N;
  const double PI = 3.14159265358979323846;
  F.L = sqrt((double)N / sqrt(2.0));
  for (int n = 1; n <= N; ++n) {
    double acc = 0.0;
    for (int k = -M + 1; k <= M - 1; ++k) {
      double theta = k * PI / M, t = F.L * tan(0.5 * theta);
      acc += exp(-t * t) * (F.L * F.L + t * t) * cos(n * theta);
    }
    F.a[N - n] = acc / (2.0 * M);
  }
}

#ifdef __CUDACC__
__device__ __forceinline__ double2 cdiv(double2 a, double2 b) {
  double inv = 1.0 / (b.x * b.x + b.y * b.y);
  return make_double2((a.x * b.x + a.y * b.y) * inv, (a.y * b.x - a.x * b.y) * inv);
}

// w(z), Im z >= 0.  The polynomial is evaluated as two interleaved Horner chains in Z^2 (odd and even powers): half the
// dependent depth of the 39-step chain.  Callers keep ONE call site per convolution (both half planes share it): ncu
// showed 33 % of tres_kernel's warp samples waiting for instruction fetch (stall_no_inst) with six inlined copies of
// the chain.  (Measured on 2 M events, all rows: six copies, one chain 142 us; this form 127 us; one out-of-line copy
// with a rolled loop 156 us.)
__device__ __forceinline__ double2 faddeeva_upper(const FaddTab &F, double2 z) {
  // i z = (-z.y, z.x)
  double2 num = make_double2(F.L - z.y, z.x), den = make_double2(F.L + z.y, -z.x);
  double2 inv = cdiv(make_double2(1.0, 0.0), den);           // 1 / (L - i z)
  double2 Z = make_double2(num.x * inv.x - num.y * inv.y, num.x * inv.y + num.y * inv.x);
  double2 Z2 = make_double2(Z.x * Z.x - Z.y * Z.y, 2.0 * Z.x * Z.y);
  // a[n] multiplies Z^(N-1-n), N even: even n -> odd powers Z * Z2^((N-2-n)/2), odd n -> even powers Z2^((N-1-n)/2)
  double2 po = make_double2(F.a[0], 0.0), pe = make_double2(F.a[1], 0.0);
#pragma unroll
  for (int n = 2; n < FADD_N; n += 2) {
    double por = fma(po.x, Z2.x, fma(-po.y, Z2.y, F.a[n])), poi = fma(po.x, Z2.y, po.y * Z2.x);
    double per = fma(pe.x, Z2.x, fma(-pe.y, Z2.y, F.a[n + 1])), pei = fma(pe.x, Z2.y, pe.y * Z2.x);
    po = make_double2(por, poi);
    pe = make_double2(per, pei);
  }
  double2 p = make_double2(fma(po.x, Z.x, fma(-po.y, Z.y, pe.x)), fma(po.x, Z.y, fma(po.y, Z.x, pe.y)));
  double2 inv2 = make_double2(inv.x * inv.x - inv.y * inv.y, 2.0 * inv.x * inv.y);
  double2 r = make_double2(p.x * inv2.x - p.y * inv2.y, p.x * inv2.y + p.y * inv2.x);
  const double RSPI = 0.56418958354775628695;                 // 1/sqrt(pi)
  return make_double2(fma(2.0, r.x, RSPI * inv.x), fma(2.0, r.y, RSPI * inv.y));
}
static_assert(FADD_N % 2 == 0, "faddeeva_upper splits the polynomial into odd and even powers");

// g0 = exp(-t^2 / (2 sigma^2)) with the two exact shortcuts of the window edges: 1 at t = 0, 0 once it underflows
__device__ __forceinline__ double gauss0(double t, double sigma) {
  if (t == 0.0) return 1.0;
  double ts = t / sigma, a = 0.5 * ts * ts;
  return a > 746.0 ? 0.0 : exp(-a);
}

// h for real lambda
__device__ __forceinline__ double conv_exp_real(double t, double lam, double sigma) {
  const double RS2 = 0.70710678118654752440;
  double u = (lam * sigma * sigma - t) * (RS2 / sigma);
  double g0 = gauss0(t, sigma);
  const bool upper = u >= 0.0;
  double E = 0.0;
  if (!upper) {
    E = exp(0.5 * lam * lam * sigma * sigma - lam * t);
    if (g0 < 1e-18 * E) return E;                             // correction below half an ulp (erfcx <= 1): same bits
  }
  const double w = erfcx(fabs(u));                            // one call site for both half planes (code size)
  return upper ? 0.5 * g0 * w : E - 0.5 * g0 * w;
}

// h for complex lambda = (lr, li)
__device__ __forceinline__ double2 conv_exp_complex(const FaddTab &F, double t, double lr, double li, double sigma) {
  const double RS2 = 0.70710678118654752440;
  double ur = (lr * sigma * sigma - t) * (RS2 / sigma), ui = li * sigma * RS2;
  double g0 = gauss0(t, sigma);
  const bool upper = ur >= 0.0;
  double mag = 0.0, sn = 0.0, cs = 0.0;
  if (!upper) {
    double s2 = sigma * sigma;
    double ere = 0.5 * (lr * lr - li * li) * s2 - lr * t, eim = lr * li * s2 - li * t;
    mag = exp(ere);
    sincos(eim, &sn, &cs);
    if (g0 < 1e-18 * mag * fmin(fabs(cs), fabs(sn))) return make_double2(mag * cs, mag * sn);   // |w| <= 1: below half an ulp
  }
  // one call site: w(i u) in the upper half plane, w(-i u) in the lower
  double2 w = faddeeva_upper(F, upper ? make_double2(-ui, ur) : make_double2(ui, -ur));
  if (upper) return make_double2(0.5 * g0 * w.x, 0.5 * g0 * w.y);
  return make_double2(mag * cs - 0.5 * g0 * w.x, mag * sn - 0.5 * g0 * w.y);
}

// window integrals int_{lo}^{hi} h dt; hi may be +inf, lo may be -inf
__device__ __forceinline__ double erf_scaled(double t, double sigma) {
  if (t == 0.0) return 0.0;
  double a = t * 0.70710678118654752440 / sigma;
  if (fabs(a) > 6.0) return a > 0.0 ? 1.0 : -1.0;            // erf(6) = 1 - 2e-17: rounds to 1 (also t = +-inf)
  return erf(a);
}
// derf = erf(hi / (sqrt2 sigma)) - erf(lo / (sqrt2 sigma)), the same for all three lambdas of an event
__device__ __forceinline__ double window_real(double lo, double hi, double lam, double sigma, double derf) {
  double hl = isinf(lo) ? 0.0 : conv_exp_real(lo, lam, sigma);
  double hh = isinf(hi) ? 0.0 : conv_exp_real(hi, lam, sigma);
  return (derf - 2.0 * (hh - hl)) / (2.0 * lam);
}
__device__ __forceinline__ double2 window_complex(const FaddTab &F, double lo, double hi, double lr, double li, double sigma,
                                                  double derf) {
  double2 hl = isinf(lo) ? make_double2(0.0, 0.0) : conv_exp_complex(F, lo, lr, li, sigma);
  double2 hh = isinf(hi) ? make_double2(0.0, 0.0) : conv_exp_complex(F, hi, lr, li, sigma);
  double2 num = make_double2(derf - 2.0 * (hh.x - hl.x), -2.0 * (hh.y - hl.y));
  return cdiv(num, make_double2(2.0 * lr, 2.0 * li));
}

// The eight per-event time quantities of one data event: psi[0..3] replace e^{-Gamma t}{cosh, cos, sinh, sin} at the
// observed time, tint[0..3] are their integrals over the window for this event's sigma.
__device__ __forceinline__ void time_terms(const FaddTab &F, double t, double sigma, double x, double y, double Gamma,
                                           double t_lo, double t_hi, double psi[4], double tint[4]) {
  double lm = Gamma * (1.0 - y), lp = Gamma * (1.0 + y), lxr = Gamma, lxi = -Gamma * x;
  double hm = conv_exp_real(t, lm, sigma), hp = conv_exp_real(t, lp, sigma);
  double2 hx = conv_exp_complex(F, t, lxr, lxi, sigma);
  psi[0] = 0.5 * (hm + hp); psi[1] = hx.x; psi[2] = 0.5 * (hm - hp); psi[3] = hx.y;
  if (tint) {
    const double derf = erf_scaled(t_hi, sigma) - erf_scaled(t_lo, sigma);
    double Im = window_real(t_lo, t_hi, lm, sigma, derf), Ip = window_real(t_lo, t_hi, lp, sigma, derf);
    double2 Ix = window_complex(F, t_lo, t_hi, lxr, lxi, sigma, derf);
    tint[0] = 0.5 * (Im + Ip); tint[1] = Ix.x; tint[2] = 0.5 * (Im - Ip); tint[3] = Ix.y;
  }
}

// The four window integrals depend on the event only through sigma, and they are smooth in it: per call (x, y, tau moved)
// one warp evaluates them exactly at TRES_NODES Chebyshev nodes of [sigma_min, sigma_max] of the data sample and turns
// the values into Chebyshev coefficients; each event then costs four short Clenshaw sums instead of four real and two
// complex convolutions at the window edges (tres_kernel: 989 -> 4xx us per 10 M events).  The table declares itself
// unusable (ok = 0: the kernel evaluates the edges exactly, as before) unless its last eight coefficients are below
// 1e-15 of the largest one, i.e. unless the interpolant has converged to rounding level on this sigma range.
// (A NaN anywhere -- sigma <= 0 -- makes every comparison fail: ok = 0.)
constexpr int TRES_NODES = 32;
struct TresTable {
  double mid, half;               // sigma = mid + half * xi, xi in [-1, 1]
  int deg, ok;                    // highest coefficient worth summing; 1: converged
  double c[4][TRES_NODES];        // Chebyshev coefficients of tint[m] (c[m][0] already halved)
};
__device__ __forceinline__ void window_terms(const FaddTab &F, double sigma, double x, double y, double Gamma, double t_lo,
                                             double t_hi, double tint[4]) {
  double lm = Gamma * (1.0 - y), lp = Gamma * (1.0 + y), lxr = Gamma, lxi = -Gamma * x;
  const double derf = erf_scaled(t_hi, sigma) - erf_scaled(t_lo, sigma);
  double Im = window_real(t_lo, t_hi, lm, sigma, derf), Ip = window_real(t_lo, t_hi, lp, sigma, derf);
  double2 Ix = window_complex(F, t_lo, t_hi, lxr, lxi, sigma, derf);
  tint[0] = 0.5 * (Im + Ip); tint[1] = Ix.x; tint[2] = 0.5 * (Im - Ip); tint[3] = Ix.y;
}
// one warp: exact values at the nodes, discrete cosine sums, convergence test
__global__ void __launch_bounds__(32) tres_table_kernel(const __grid_constant__ FaddTab F, double x, double y, double Gamma,
                                                        double t_lo, double t_hi, double sig_lo, double sig_hi,
                                                        TresTable *__restrict__ out) {
  const int lane = threadIdx.x;
  const double mid = 0.5 * (sig_lo + sig_hi), half = 0.5 * (sig_hi - sig_lo);
  double f[4];
  window_terms(F, mid + half * cospi((lane + 0.5) / TRES_NODES), x, y, Gamma, t_lo, t_hi, f);
  double c[4] = {0.0, 0.0, 0.0, 0.0};
  for (int j = 0; j < TRES_NODES; ++j) {
    const double w = cospi(lane * (j + 0.5) / TRES_NODES);
#pragma unroll
    for (int m = 0; m < 4; ++m) c[m] = fma(__shfl_sync(0xffffffffu, f[m], j), w, c[m]);
  }
  // one scale for all four series: tint[2], tint[3] are differences of quantities of the size of tint[0] and carry its
  // rounding noise, in the exact evaluation as much as here
  double mx = 0.0;
#pragma unroll
  for (int m = 0; m < 4; ++m) {
    c[m] *= (lane == 0 ? 1.0 : 2.0) / TRES_NODES;
    mx = fmax(mx, fabs(c[m]));
    out->c[m][lane] = c[m];
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  bool small = true;
#pragma unroll
  for (int m = 0; m < 4; ++m) small = small && fabs(c[m]) <= 1e-15 * mx;
  const unsigned big = __ballot_sync(0xffffffffu, !small);            // lanes = orders that still matter
  const bool ok = (big >> (TRES_NODES - 8)) == 0u && isfinite(mx) && sig_lo > 0.0;   // sigma_t <= 0 is outside the contract: the exact path reports it
  const int deg = big ? 31 - __clz(big) : 0;
  if (lane == 0) { out->mid = mid; out->half = half; out->deg = deg; out->ok = ok ? 1 : 0; }
}
// Clenshaw sums of the four series at one sigma; tab: the table in shared memory
__device__ __forceinline__ void window_terms_table(const TresTable &tab, double sigma, double tint[4]) {
  const double xi = tab.half > 0.0 ? (sigma - tab.mid) / tab.half : 0.0, x2 = 2.0 * xi;
  double b1[4] = {0.0, 0.0, 0.0, 0.0}, b2[4] = {0.0, 0.0, 0.0, 0.0};
  for (int k = tab.deg; k >= 1; --k) {
#pragma unroll
    for (int m = 0; m < 4; ++m) {
      double b0 = fma(x2, b1[m], tab.c[m][k] - b2[m]);
      b2[m] = b1[m]; b1[m] = b0;
    }
  }
#pragma unroll
  for (int m = 0; m < 4; ++m) tint[m] = fma(xi, b1[m], tab.c[m][0] - b2[m]);
}

// Derivatives with respect to the mixing parameters (tddp4_nll_grad in resolution mode).  From the definition,
//   dh/dlambda = (lambda sigma^2 - t) h - sigma g0 / sqrt(2 pi),      dH/dlambda = -H/lambda - (dh/dlambda)/lambda,
// and d lambda_-+ / dy = -+Gamma, d lambda_x / dx = -i Gamma.  out[0..3] = d psi_1/dx, d psi_3/dx, d psi_0/dy, d psi_2/dy;
// out[4..7] = d T_1/dx, d T_3/dx, d T_0/dy, d T_2/dy (the other derivatives vanish).
__device__ __forceinline__ double dconv_real(double t, double lam, double sigma, double h) {
  return (lam * sigma * sigma - t) * h - sigma * gauss0(t, sigma) * 0.39894228040143267794;   // 1/sqrt(2 pi)
}
__device__ __forceinline__ double2 dconv_complex(double t, double lr, double li, double sigma, double2 h) {
  double ar = lr * sigma * sigma - t, ai = li * sigma * sigma;
  return make_double2(ar * h.x - ai * h.y - sigma * gauss0(t, sigma) * 0.39894228040143267794, ar * h.y + ai * h.x);
}
__device__ __forceinline__ void time_term_derivatives(const FaddTab &F, double t, double sigma, double x, double y, double Gamma,
                                                      double t_lo, double t_hi, double out[8]) {
  const double lm = Gamma * (1.0 - y), lp = Gamma * (1.0 + y), lxr = Gamma, lxi = -Gamma * x;
  // at the observed time
  double dm = dconv_real(t, lm, sigma, conv_exp_real(t, lm, sigma));
  double dp = dconv_real(t, lp, sigma, conv_exp_real(t, lp, sigma));
  double2 dx = dconv_complex(t, lxr, lxi, sigma, conv_exp_complex(F, t, lxr, lxi, sigma));
  out[0] = Gamma * dx.y;  out[1] = -Gamma * dx.x;              // -i Gamma (a + i b) = Gamma b - i Gamma a
  out[2] = 0.5 * Gamma * (dp - dm);  out[3] = -0.5 * Gamma * (dp + dm);
  // window integrals: dI/dlambda = -I/lambda - (dh(hi) - dh(lo))/lambda
  const double derf = erf_scaled(t_hi, sigma) - erf_scaled(t_lo, sigma);
  auto edge_real = [&](double lam) {
    double hl = isinf(t_lo) ? 0.0 : conv_exp_real(t_lo, lam, sigma), hh = isinf(t_hi) ? 0.0 : conv_exp_real(t_hi, lam, sigma);
    double I = (derf - 2.0 * (hh - hl)) / (2.0 * lam);
    double dl = isinf(t_lo) ? 0.0 : dconv_real(t_lo, lam, sigma, hl), dh = isinf(t_hi) ? 0.0 : dconv_real(t_hi, lam, sigma, hh);
    return -(I + (dh - dl)) / lam;
  };
  double Dm = edge_real(lm), Dp = edge_real(lp);
  double2 hl = isinf(t_lo) ? make_double2(0.0, 0.0) : conv_exp_complex(F, t_lo, lxr, lxi, sigma);
  double2 hh = isinf(t_hi) ? make_double2(0.0, 0.0) : conv_exp_complex(F, t_hi, lxr, lxi, sigma);
  double2 I = cdiv(make_double2(derf - 2.0 * (hh.x - hl.x), -2.0 * (hh.y - hl.y)), make_double2(2.0 * lxr, 2.0 * lxi));
  double2 dl = isinf(t_lo) ? make_double2(0.0, 0.0) : dconv_complex(t_lo, lxr, lxi, sigma, hl);
  double2 dh = isinf(t_hi) ? make_double2(0.0, 0.0) : dconv_complex(t_hi, lxr, lxi, sigma, hh);
  double2 Dx = cdiv(make_double2(-(I.x + dh.x - dl.x), -(I.y + dh.y - dl.y)), make_double2(lxr, lxi));
  out[4] = Gamma * Dx.y;  out[5] = -Gamma * Dx.x;
  out[6] = 0.5 * Gamma * (Dp - Dm);  out[7] = -0.5 * Gamma * (Dp + Dm);
}
#endif  // __CUDACC__

}  // namespace tddp4k
