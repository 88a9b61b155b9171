// grad_kernels.cuh -- NLL and its analytic gradient with respect to the couplings and the mixing parameters in ONE pass
// over the cached coupling columns.  A gradient-based host minimiser otherwise needs 2 (4 K_c + 2)
// NLL evaluations per gradient.
//
// With gA = dB/dA* = (cosh+cos) A - (sinh + i sin) Abar and gAbar = dB/dAbar* = (cosh-cos) Abar - (sinh - i sin) A (B the
// bracket of eq. (1); A = sum_k c_k a_k, eq. (2)):
//     dB/dRe c_k = 2 Re(conj(gA) a_k),   dB/dIm c_k = -2 Im(conj(gA) a_k),   likewise for cbar with gAbar,
//     dB/dx = Gamma t [-(|A|^2-|Abar|^2) sin - 2 Im(A Abar*) cos],   dB/dy = Gamma t [(|A|^2+|Abar|^2) sinh - 2 Re(A Abar*) cosh].
// The kernel accumulates D_k = sum_i conj(gA_i) a_ik / B_i, Dbar_k, sum_i (dB_i/dx)/B_i, sum_i (dB_i/dy)/B_i next to
// sum_i log B_i; the last block adds the normalisation part from the Gram matrix in force (Hermitian G, u = c^T G / n,
// ubar = cbar^T G / n):   dN/dc_k* = (T0+T1) u_k - (T2 + i T3) ubar_k,   dN/dcbar_k* = (T0-T1) ubar_k - (T2 - i T3) u_k,
//     dN/dx = T1' (nAA - nBB) - 2 T3' Im X,   dN/dy = T0' (nAA + nBB) - 2 T2' Re X,
// and writes  grad = -(data part) + n (dN/dtheta) / N.   Deterministic: fixed-order block and grid reductions.
#pragma once

namespace tddp4k {

struct GradParams {
  double dT1dx, dT3dx, dT0dy, dT2dy;   // derivatives of the time integrals (host, closed form)
};

// result layout: [0..4] as the NLL kernels (sum log B, sum t, N, NLL, #bad), [8 ...] the 4 K_c + 2 gradient entries
constexpr int GRAD_OFFSET = 8;

template <int KC, bool SMALL>
__global__ void __launch_bounds__(STREAM_BLOCK, KC <= 8 ? 2 : 1)
nll_grad_kernel(const double2 *__restrict__ a, const double *__restrict__ t, int64_t ld, int64_t n,
                const __grid_constant__ RateParams R, const __grid_constant__ GradParams GP, const double *__restrict__ G,
                double inv_n_norm, double sum_t, double *__restrict__ partials /* [grid][NA + 3] */, unsigned int *ticket,
                double *__restrict__ result) {
  constexpr int NA = 4 * KC + 2, PS = NA + 3;
  __shared__ double s_red[STREAM_WARPS][NA];
  __shared__ double s_sum[NA];
  __shared__ double s_p[STREAM_WARPS];
  __shared__ long long s_e[STREAM_WARPS];
  __shared__ int s_b[STREAM_WARPS];
  __shared__ double s_n[4];
  __shared__ double2 s_u[KC], s_ub[KC];
  __shared__ bool last;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  MantAcc la;
  double acc[NA];
#pragma unroll
  for (int j = 0; j < NA; ++j) acc[j] = 0.0;
  const double yG = R.y * R.Gamma, xG = R.x * R.Gamma;
  const int64_t stride = (int64_t)gridDim.x * STREAM_BLOCK;
#pragma unroll 1
  for (int64_t i = (int64_t)blockIdx.x * STREAM_BLOCK + tid; i < n; i += stride) {
    double2 v[KC];
#pragma unroll
    for (int c = 0; c < KC; ++c) v[c] = ldg_stream2(a + c * ld + i);
    const double ti = ldg_stream1(t + i);
    double2 A = make_double2(0.0, 0.0), Ab = make_double2(0.0, 0.0);
#pragma unroll
    for (int c = 0; c < KC; ++c) amp_add(A, Ab, R.c[c][0], R.c[c][1], R.cbar[c][0], R.cbar[c][1], v[c]);
    double ch, sh, cs, sn;
    mixing_functions<SMALL>(yG * ti, xG * ti, ch, sh, cs, sn);
    const Bilinears q = bilinears(A, Ab);
    const double aa = q.aa, bb = q.bb, cre = q.cre, cim = q.cim;
    const double B = rate_form(q, ch, cs, sh, sn);                                        // the bits of bracket()
    la.add(B);
    const double inv = 1.0 / B;
    const double gx = ((ch + cs) * A.x - (sh * Ab.x - sn * Ab.y)) * inv, gy = ((ch + cs) * A.y - (sh * Ab.y + sn * Ab.x)) * inv;
    const double hx = ((ch - cs) * Ab.x - (sh * A.x + sn * A.y)) * inv, hy = ((ch - cs) * Ab.y - (sh * A.y - sn * A.x)) * inv;
#pragma unroll
    for (int c = 0; c < KC; ++c) {
      acc[2 * c] = fma(gx, v[c].x, fma(gy, v[c].y, acc[2 * c]));                 // Re conj(gA) a_c
      acc[2 * c + 1] = fma(gx, v[c].y, fma(-gy, v[c].x, acc[2 * c + 1]));         // Im conj(gA) a_c
      acc[2 * KC + 2 * c] = fma(hx, v[c].x, fma(hy, v[c].y, acc[2 * KC + 2 * c]));
      acc[2 * KC + 2 * c + 1] = fma(hx, v[c].y, fma(-hy, v[c].x, acc[2 * KC + 2 * c + 1]));
    }
    const double gt = R.Gamma * ti * inv;
    acc[4 * KC] += gt * (-(aa - bb) * sn - 2.0 * cim * cs);
    acc[4 * KC + 1] += gt * ((aa + bb) * sh - 2.0 * cre * ch);
  }
  // block partials, fixed order: lanes by butterfly, warps in index order
#pragma unroll
  for (int j = 0; j < NA; ++j) {
    double s = warp_sum(acc[j]);
    if (lane == 0) s_red[warp][j] = s;
  }
  warp_merge(la);
  if (lane == 0) { s_p[warp] = la.prod; s_e[warp] = la.esum; s_b[warp] = la.bad; }
  __syncthreads();
  double *mine = partials + (int64_t)blockIdx.x * PS;
  for (int j = tid; j < NA; j += STREAM_BLOCK) {
    double s = 0.0;
#pragma unroll
    for (int w = 0; w < STREAM_WARPS; ++w) s += s_red[w][j];
    mine[j] = s;
  }
  if (tid == 0) {
    MantAcc m;
#pragma unroll
    for (int w = 0; w < STREAM_WARPS; ++w) m.merge(s_p[w], s_e[w], s_b[w]);
    m.renorm();
    mine[NA] = m.prod; mine[NA + 1] = (double)m.esum; mine[NA + 2] = (double)m.bad;
  }
  __threadfence();
  __syncthreads();
  if (tid == 0) last = atomicAdd(ticket, 1u) == gridDim.x - 1;
  __syncthreads();
  if (!last) return;
  __threadfence();
  // last block: sums over blocks (16 chains per entry, fixed tree), mantissa products merged in block order by warp 0
  for (int j = tid; j < NA; j += STREAM_BLOCK) {
    double part[16];
#pragma unroll
    for (int c = 0; c < 16; ++c) part[c] = 0.0;
    for (unsigned b = 0; b < gridDim.x; b += 16) {
#pragma unroll
      for (int c = 0; c < 16; ++c)
        if (b + c < gridDim.x) part[c] += __ldcg(partials + (int64_t)(b + c) * PS + j);
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < 16; ++c) s += part[c];
    s_sum[j] = s;
  }
  MantAcc m;
  if (warp == STREAM_WARPS - 1) {
    for (unsigned b = lane; b < gridDim.x; b += 32) {
      const double *pb = partials + (int64_t)b * PS + NA;
      m.merge(__ldcg(pb), (long long)__ldcg(pb + 1), (int)__ldcg(pb + 2));
      m.renorm();
    }
    warp_merge(m);
    if (lane == 0) { s_p[0] = m.prod; s_e[0] = m.esum; s_b[0] = m.bad; }
  } else if (warp == 1) {
    double nAA, nBB, xr, xi;
    gram_sums_warp(R, G, KC, inv_n_norm, nAA, nBB, xr, xi);
    if (lane == 0) { s_n[0] = nAA; s_n[1] = nBB; s_n[2] = xr; s_n[3] = xi; }
  } else if (warp == 2 && lane < KC) {
    double2 u = make_double2(0.0, 0.0), ub = make_double2(0.0, 0.0);   // u_k = sum_j c_j G_jk / n, ubar_k with cbar
    for (int j = 0; j < KC; ++j) {
      double gr = __ldcg(G + (j * KC + lane) * 2) * inv_n_norm, gi = __ldcg(G + (j * KC + lane) * 2 + 1) * inv_n_norm;
      u.x += R.c[j][0] * gr - R.c[j][1] * gi;    u.y += R.c[j][0] * gi + R.c[j][1] * gr;
      ub.x += R.cbar[j][0] * gr - R.cbar[j][1] * gi;  ub.y += R.cbar[j][0] * gi + R.cbar[j][1] * gr;
    }
    s_u[lane] = u; s_ub[lane] = ub;
  }
  __syncthreads();
  const double nAA = s_n[0], nBB = s_n[1], xr = s_n[2], xi = s_n[3];
  const double norm = R.T[0] * (nAA + nBB) + R.T[1] * (nAA - nBB) - 2.0 * R.T[2] * xr - 2.0 * R.T[3] * xi;
  const double scale = (double)n / norm;
  if (tid < KC) {
    const double2 u = s_u[tid], ub = s_ub[tid];
    // h = (T0+T1) u - (T2 + i T3) ubar;  hbar = (T0-T1) ubar - (T2 - i T3) u
    const double hr = (R.T[0] + R.T[1]) * u.x - (R.T[2] * ub.x - R.T[3] * ub.y);
    const double hi = (R.T[0] + R.T[1]) * u.y - (R.T[2] * ub.y + R.T[3] * ub.x);
    const double br = (R.T[0] - R.T[1]) * ub.x - (R.T[2] * u.x + R.T[3] * u.y);
    const double bi = (R.T[0] - R.T[1]) * ub.y - (R.T[2] * u.y - R.T[3] * u.x);
    double *g = result + GRAD_OFFSET;
    g[2 * tid] = -2.0 * s_sum[2 * tid] + scale * 2.0 * hr;
    g[2 * tid + 1] = 2.0 * s_sum[2 * tid + 1] + scale * 2.0 * hi;
    g[2 * KC + 2 * tid] = -2.0 * s_sum[2 * KC + 2 * tid] + scale * 2.0 * br;
    g[2 * KC + 2 * tid + 1] = 2.0 * s_sum[2 * KC + 2 * tid + 1] + scale * 2.0 * bi;
  }
  if (tid == 0) {
    double *g = result + GRAD_OFFSET;
    g[4 * KC] = -s_sum[4 * KC] + scale * (GP.dT1dx * (nAA - nBB) - 2.0 * GP.dT3dx * xi);
    g[4 * KC + 1] = -s_sum[4 * KC + 1] + scale * (GP.dT0dy * (nAA + nBB) - 2.0 * GP.dT2dy * xr);
    const double prod = s_p[0];
    const long long esum = s_e[0];
    const int bad = s_b[0];
    double s0 = log(prod) + 0.693147180559945309417 * (double)esum;
    double nll = R.Gamma * sum_t - s0 + (double)n * log(norm);
    if (bad > 0 || !(norm > 0.0)) nll = INFINITY;
    result[0] = s0; result[1] = sum_t; result[2] = norm; result[3] = nll; result[4] = (double)bad;
    *ticket = 0;
  }
}

// ------------------------------------------------------------------------------------------------
// The same in resolution mode (config 5): P_i = R_i / N_i with R_i the bracket with the convolved time functions psi_m of
// the event and N_i = sum_m T_m(sigma_i) S_m (stream_kernels.cuh, resolved_prob).  Per event the kernel reads the K_c
// columns, the eight time rows and the eight derivative rows (tres_grad_kernel).  d(sum log N_i)/dc_k* keeps the Gram
// structure with per-call weights W_m = sum_i T_m,i / N_i:  (W0+W1) u_k - (W2 + i W3) ubar_k.
template <int KC>
__global__ void __launch_bounds__(STREAM_BLOCK, 1)
nll_grad_res_kernel(const double2 *__restrict__ a, const double *__restrict__ tr, const double *__restrict__ trg, int64_t ld,
                    int64_t n, const __grid_constant__ RateParams R, const double *__restrict__ G, double inv_n_norm,
                    double *__restrict__ partials /* [grid][NA + 3] */, unsigned int *ticket, double *__restrict__ result) {
  constexpr int NG = 4 * KC + 2, NA = NG + 4, PS = NA + 3;
  __shared__ double s_red[STREAM_WARPS][NA];
  __shared__ double s_sum[NA];
  __shared__ double s_p[STREAM_WARPS];
  __shared__ long long s_e[STREAM_WARPS];
  __shared__ int s_b[STREAM_WARPS];
  __shared__ double s_S[4];
  __shared__ double2 s_u[KC], s_ub[KC];
  __shared__ bool last;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  block_phase_space_sums(R, G, KC, inv_n_norm, s_S);
  const double S1 = s_S[0], S2 = s_S[1], S3 = s_S[2], S4 = s_S[3];
  MantAcc la;
  double acc[NA];
#pragma unroll
  for (int j = 0; j < NA; ++j) acc[j] = 0.0;
  const int64_t stride = (int64_t)gridDim.x * STREAM_BLOCK;
#pragma unroll 1
  for (int64_t i = (int64_t)blockIdx.x * STREAM_BLOCK + tid; i < n; i += stride) {
    double2 v[KC];
    double w[8], d[8];
#pragma unroll
    for (int c = 0; c < KC; ++c) v[c] = ldg_stream2(a + c * ld + i);
#pragma unroll
    for (int m = 0; m < 8; ++m) { w[m] = ldg_stream1(tr + m * ld + i); d[m] = ldg_stream1(trg + m * ld + i); }
    double2 A = make_double2(0.0, 0.0), Ab = make_double2(0.0, 0.0);
#pragma unroll
    for (int c = 0; c < KC; ++c) amp_add(A, Ab, R.c[c][0], R.c[c][1], R.cbar[c][0], R.cbar[c][1], v[c]);
    const Bilinears q = bilinears(A, Ab);
    const double aa = q.aa, bb = q.bb, cre = q.cre, cim = q.cim;
    const double Rv = rate_form(q, w[0], w[1], w[2], w[3]);                                        // the bits of resolved_prob()
    const double Nv = fma(S1, w[4], fma(S2, w[5], fma(-2.0 * S3, w[6], __dmul_rn(-2.0 * S4, w[7]))));
    la.add(__ddiv_rn(Rv, Nv));
    const double invR = 1.0 / Rv, invN = 1.0 / Nv;
    const double gx = ((w[0] + w[1]) * A.x - (w[2] * Ab.x - w[3] * Ab.y)) * invR, gy = ((w[0] + w[1]) * A.y - (w[2] * Ab.y + w[3] * Ab.x)) * invR;
    const double hx = ((w[0] - w[1]) * Ab.x - (w[2] * A.x + w[3] * A.y)) * invR, hy = ((w[0] - w[1]) * Ab.y - (w[2] * A.y - w[3] * A.x)) * invR;
#pragma unroll
    for (int c = 0; c < KC; ++c) {
      acc[2 * c] = fma(gx, v[c].x, fma(gy, v[c].y, acc[2 * c]));
      acc[2 * c + 1] = fma(gx, v[c].y, fma(-gy, v[c].x, acc[2 * c + 1]));
      acc[2 * KC + 2 * c] = fma(hx, v[c].x, fma(hy, v[c].y, acc[2 * KC + 2 * c]));
      acc[2 * KC + 2 * c + 1] = fma(hx, v[c].y, fma(-hy, v[c].x, acc[2 * KC + 2 * c + 1]));
    }
    // d log(R/N) / dx, / dy: d = (dpsi1/dx, dpsi3/dx, dpsi0/dy, dpsi2/dy, dT1/dx, dT3/dx, dT0/dy, dT2/dy)
    acc[4 * KC] += ((aa - bb) * d[0] - 2.0 * cim * d[1]) * invR - (S2 * d[4] - 2.0 * S4 * d[5]) * invN;
    acc[4 * KC + 1] += ((aa + bb) * d[2] - 2.0 * cre * d[3]) * invR - (S1 * d[6] - 2.0 * S3 * d[7]) * invN;
#pragma unroll
    for (int m = 0; m < 4; ++m) acc[NG + m] = fma(w[4 + m], invN, acc[NG + m]);     // W_m
  }
#pragma unroll
  for (int j = 0; j < NA; ++j) {
    double s = warp_sum(acc[j]);
    if (lane == 0) s_red[warp][j] = s;
  }
  warp_merge(la);
  if (lane == 0) { s_p[warp] = la.prod; s_e[warp] = la.esum; s_b[warp] = la.bad; }
  __syncthreads();
  double *mine = partials + (int64_t)blockIdx.x * PS;
  for (int j = tid; j < NA; j += STREAM_BLOCK) {
    double s = 0.0;
#pragma unroll
    for (int wp = 0; wp < STREAM_WARPS; ++wp) s += s_red[wp][j];
    mine[j] = s;
  }
  if (tid == 0) {
    MantAcc m;
#pragma unroll
    for (int wp = 0; wp < STREAM_WARPS; ++wp) m.merge(s_p[wp], s_e[wp], s_b[wp]);
    m.renorm();
    mine[NA] = m.prod; mine[NA + 1] = (double)m.esum; mine[NA + 2] = (double)m.bad;
  }
  __threadfence();
  __syncthreads();
  if (tid == 0) last = atomicAdd(ticket, 1u) == gridDim.x - 1;
  __syncthreads();
  if (!last) return;
  __threadfence();
  for (int j = tid; j < NA; j += STREAM_BLOCK) {
    double part[16];
#pragma unroll
    for (int c = 0; c < 16; ++c) part[c] = 0.0;
    for (unsigned b = 0; b < gridDim.x; b += 16) {
#pragma unroll
      for (int c = 0; c < 16; ++c)
        if (b + c < gridDim.x) part[c] += __ldcg(partials + (int64_t)(b + c) * PS + j);
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < 16; ++c) s += part[c];
    s_sum[j] = s;
  }
  if (warp == STREAM_WARPS - 1) {
    MantAcc m;
    for (unsigned b = lane; b < gridDim.x; b += 32) {
      const double *pb = partials + (int64_t)b * PS + NA;
      m.merge(__ldcg(pb), (long long)__ldcg(pb + 1), (int)__ldcg(pb + 2));
      m.renorm();
    }
    warp_merge(m);
    if (lane == 0) { s_p[0] = m.prod; s_e[0] = m.esum; s_b[0] = m.bad; }
  } else if (warp == 2 && lane < KC) {
    double2 u = make_double2(0.0, 0.0), ub = make_double2(0.0, 0.0);
    for (int j = 0; j < KC; ++j) {
      double gr = __ldcg(G + (j * KC + lane) * 2) * inv_n_norm, gi = __ldcg(G + (j * KC + lane) * 2 + 1) * inv_n_norm;
      u.x += R.c[j][0] * gr - R.c[j][1] * gi;    u.y += R.c[j][0] * gi + R.c[j][1] * gr;
      ub.x += R.cbar[j][0] * gr - R.cbar[j][1] * gi;  ub.y += R.cbar[j][0] * gi + R.cbar[j][1] * gr;
    }
    s_u[lane] = u; s_ub[lane] = ub;
  }
  __syncthreads();
  const double W0 = s_sum[NG], W1 = s_sum[NG + 1], W2 = s_sum[NG + 2], W3 = s_sum[NG + 3];
  double *g = result + GRAD_OFFSET;
  if (tid < KC) {
    const double2 u = s_u[tid], ub = s_ub[tid];
    const double hr = (W0 + W1) * u.x - (W2 * ub.x - W3 * ub.y), hi = (W0 + W1) * u.y - (W2 * ub.y + W3 * ub.x);
    const double br = (W0 - W1) * ub.x - (W2 * u.x + W3 * u.y), bi = (W0 - W1) * ub.y - (W2 * u.y - W3 * u.x);
    g[2 * tid] = -2.0 * s_sum[2 * tid] + 2.0 * hr;
    g[2 * tid + 1] = 2.0 * s_sum[2 * tid + 1] + 2.0 * hi;
    g[2 * KC + 2 * tid] = -2.0 * s_sum[2 * KC + 2 * tid] + 2.0 * br;
    g[2 * KC + 2 * tid + 1] = 2.0 * s_sum[2 * KC + 2 * tid + 1] + 2.0 * bi;
  }
  if (tid == 0) {
    g[4 * KC] = -s_sum[4 * KC];
    g[4 * KC + 1] = -s_sum[4 * KC + 1];
    const double s0 = log(s_p[0]) + 0.693147180559945309417 * (double)s_e[0];
    const double norm = R.T[0] * S1 + R.T[1] * S2 - 2.0 * R.T[2] * S3 - 2.0 * R.T[3] * S4;
    double nll = -s0;
    if (s_b[0] > 0 || !(norm > 0.0)) nll = INFINITY;
    result[0] = s0; result[1] = 0.0; result[2] = norm; result[3] = nll; result[4] = (double)s_b[0];
    *ticket = 0;
  }
}

}  // namespace tddp4k
