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
//
// The 4 K_c coupling sums are ONE dense contraction over events, D = W^T X with W_i = (Re gA, Im gA, Re gAbar, Im gAbar)_i / B_i
// and X_i = (Re a_i0, Im a_i0, Re a_i1, ...): it runs on the fp64 tensor cores (mma.sync m8n8k4, SASS DMMA), 4 events per
// instruction, from per-warp shared-memory tiles laid out as in the Gram kernel (conflict-free stores and fragment loads).
// A thread then carries 2 NB accumulator registers instead of 4 K_c + 2 (the scalar form held 34 accumulators next to the
// 8 columns of its event and spilled: 31 STL / 26 LDL in the loop at 128 registers, 58.7 us per 1 M events, 0.35 of the
// HBM roofline).
#pragma once

namespace tddp4k {

struct GradParams {
  double dT1dx, dT3dx, dT0dy, dT2dy;   // derivatives of the time integrals (host, closed form)
};

// result layout: [0..4] as the NLL kernels (sum log B, sum t, N, NLL, #bad), [8 ...] the 4 K_c + 2 gradient entries
constexpr int GRAD_OFFSET = 8;

// shared-memory tiles of one warp: X [32][gram_stride(NB)] (event-major, as the Gram kernel), W [32][GRAD_WS] (rows 4..7 zero)
constexpr int GRAD_WS = 10;
// resident blocks per SM: three (24 warps, 80 registers, no spills once the grid reduction went two-level) where the
// per-warp tiles leave room, else two.  Measured at K_c = 8, 1 M events: 47 us at two blocks, 44 us at three.
template <int KC> __host__ __device__ constexpr int grad_nb() { return (KC + 3) / 4; }
template <int KC> __host__ __device__ constexpr int grad_bps() { return grad_nb<KC>() <= 2 ? 3 : 2; }
template <int KC> __host__ __device__ constexpr size_t grad_warp_bytes() {
  return align_up((size_t)32 * gram_stride(grad_nb<KC>()) * sizeof(double), 128) + align_up((size_t)32 * GRAD_WS * sizeof(double), 128);
}
template <int KC> inline size_t grad_smem_bytes() { return STREAM_WARPS * grad_warp_bytes<KC>(); }

// D += W^T X over the warp's 32 events: acc[b] holds the C fragment of feature block b (row = weight lane >> 2,
// columns 2 (lane & 3) + {0, 1}); group g takes the events 8 (g >> 1) + 2 (lane & 3) + (g & 1) (bank-conflict free)
template <int NB>
__device__ __forceinline__ void grad_mma_tile(const double *Xs, const double *Ws, double (&acc)[NB][2]) {
  constexpr int XS = gram_stride(NB);
  const int lane = threadIdx.x & 31;
  __syncwarp();
  const double *xb = Xs + (2 * (lane & 3)) * XS + (lane >> 2);
  const double *wb = Ws + (2 * (lane & 3)) * GRAD_WS + (lane >> 2);
#pragma unroll
  for (int grp = 0; grp < 8; ++grp) {
    const int e0 = 8 * (grp >> 1) + (grp & 1);
    const double w = wb[e0 * GRAD_WS];
#pragma unroll
    for (int b = 0; b < NB; ++b) dmma884(acc[b][0], acc[b][1], w, xb[e0 * XS + 8 * b]);
  }
  __syncwarp();
}

// Block and grid reduction of the gradient sums.  Per block: NB * 32 tensor-core sums C_b[m][n] (m < 4 weights, n < 8
// features), NS scalar sums, the mantissa product.  Returns true in the last block, with the grid totals in s_sum
// ([NB * 32 + NS]) and the merged product in s_p[0], s_e[0], s_b[0].
template <int NB, int NS>
__device__ __forceinline__ bool grad_reduce(double (&acc)[NB][2], double (&sc)[NS], MantAcc la, double *__restrict__ partials,
                                            unsigned int *ticket, double *s_red /* [WARPS][NB*32+NS] */, double *s_sum,
                                            double *s_p, long long *s_e, int *s_b, bool *last) {
  constexpr int NC = NB * 32, NA = NC + NS, PS = NA + 3;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (lane < 16) {
#pragma unroll
    for (int b = 0; b < NB; ++b) {
      s_red[warp * NA + b * 32 + (lane >> 2) * 8 + 2 * (lane & 3)] = acc[b][0];
      s_red[warp * NA + b * 32 + (lane >> 2) * 8 + 2 * (lane & 3) + 1] = acc[b][1];
    }
  }
#pragma unroll
  for (int j = 0; j < NS; ++j) {
    double v = warp_sum(sc[j]);
    if (lane == 0) s_red[warp * NA + NC + j] = v;
  }
  warp_merge(la);
  if (lane == 0) { s_p[warp] = la.prod; s_e[warp] = la.esum; s_b[warp] = la.bad; }
  __syncthreads();
  double *mine = partials + (int64_t)blockIdx.x * PS;
  for (int j = tid; j < NA; j += STREAM_BLOCK) {
    double v = 0.0;
#pragma unroll
    for (int w = 0; w < STREAM_WARPS; ++w) v += s_red[w * NA + j];
    mine[j] = v;
  }
  if (tid == 0) {
    MantAcc m;
#pragma unroll
    for (int w = 0; w < STREAM_WARPS; ++w) m.merge(s_p[w], s_e[w], s_b[w]);
    m.renorm();
    mine[NA] = m.prod; mine[NA + 1] = (double)m.esum; mine[NA + 2] = (double)m.bad;
  }
  // Two-level, fixed-order reduction over the grid (as the Gram kernel's, jit_shared.cuh): blocks form groups of GRAM_GROUP
  // consecutive blocks; the last block of a group to arrive adds the group's partials in block order, the last group to
  // finish adds the group sums in group order.  Every level is one round of independent loads.  (The single-level form --
  // one block pulling gridDim.x x PS doubles, 163 KB at K_c = 8, through one SM in five rounds -- left the SMs idle for a
  // third of the launch: ncu sm__cycles_active 61 k of 91 k elapsed cycles at 1 M events.)
  const unsigned n_groups = (gridDim.x + GRAM_GROUP - 1) / GRAM_GROUP, grp = blockIdx.x / GRAM_GROUP;
  const unsigned g_first = grp * GRAM_GROUP, g_size = min((unsigned)GRAM_GROUP, gridDim.x - g_first);
  double *gsum = partials + (int64_t)gridDim.x * PS;               // [n_groups][PS]
  __threadfence();
  __syncthreads();
  if (tid == 0) *last = atomicAdd(ticket + 1 + grp, 1u) == g_size - 1;
  __syncthreads();
  if (!*last) return false;
  __threadfence();
  for (int j = tid; j < NA; j += STREAM_BLOCK) {
    double v[GRAM_GROUP];
#pragma unroll
    for (int c = 0; c < GRAM_GROUP; ++c) v[c] = (unsigned)c < g_size ? __ldcg(partials + (int64_t)(g_first + c) * PS + j) : 0.0;
    double sum = 0.0;
#pragma unroll
    for (int c = 0; c < GRAM_GROUP; ++c) sum += v[c];
    gsum[(int64_t)grp * PS + j] = sum;
  }
  if (warp == STREAM_WARPS - 1) {                                  // the group's mantissa product: one lane per block
    MantAcc m;
    if ((unsigned)lane < g_size) {
      const double *src = partials + (int64_t)(g_first + lane) * PS + NA;
      m.merge(__ldcg(src), (long long)__ldcg(src + 1), (int)__ldcg(src + 2));
    }
    warp_merge(m);
    if (lane == 0) { double *dst = gsum + (int64_t)grp * PS + NA; dst[0] = m.prod; dst[1] = (double)m.esum; dst[2] = (double)m.bad; }
  }
  __threadfence();
  __syncthreads();
  if (tid == 0) { ticket[1 + grp] = 0; *last = atomicAdd(ticket, 1u) == n_groups - 1; }
  __syncthreads();
  if (!*last) return false;
  __threadfence();
  for (int j = tid; j < NA; j += STREAM_BLOCK) {
    double sum = 0.0;
    unsigned g = 0;
    for (; g + 8 <= n_groups; g += 8) {
      double v[8];
#pragma unroll
      for (int c = 0; c < 8; ++c) v[c] = __ldcg(gsum + (int64_t)(g + c) * PS + j);
#pragma unroll
      for (int c = 0; c < 8; ++c) sum += v[c];
    }
    for (; g < n_groups; ++g) sum += __ldcg(gsum + (int64_t)g * PS + j);
    s_sum[j] = sum;
  }
  if (warp == STREAM_WARPS - 1) {
    MantAcc m;
    for (unsigned g = lane; g < n_groups; g += 32) {
      const double *src = gsum + (int64_t)g * PS + NA;
      m.merge(__ldcg(src), (long long)__ldcg(src + 1), (int)__ldcg(src + 2));
      m.renorm();
    }
    warp_merge(m);
    if (lane == 0) { s_p[0] = m.prod; s_e[0] = m.esum; s_b[0] = m.bad; }
  }
  return true;
}
// sum_i W_i[m] X_i[f] from the reduced tiles
__device__ __forceinline__ double grad_c(const double *s_sum, int m, int f) { return s_sum[(f >> 3) * 32 + m * 8 + (f & 7)]; }
// u_k = sum_j c_j G_jk / n and ubar_k (Hermitian G): one lane per k
template <int KC>
__device__ __forceinline__ void grad_gram_vectors(const RateParams &R, const double *__restrict__ G, double inv_n_norm, int lane,
                                                  double2 *s_u, double2 *s_ub) {
  if (lane < KC) {
    double2 u = make_double2(0.0, 0.0), ub = make_double2(0.0, 0.0);
    for (int j = 0; j < KC; ++j) {
      double gr = __ldcg(G + (j * KC + lane) * 2) * inv_n_norm, gi = __ldcg(G + (j * KC + lane) * 2 + 1) * inv_n_norm;
      u.x += R.c[j][0] * gr - R.c[j][1] * gi;    u.y += R.c[j][0] * gi + R.c[j][1] * gr;
      ub.x += R.cbar[j][0] * gr - R.cbar[j][1] * gi;  ub.y += R.cbar[j][0] * gi + R.cbar[j][1] * gr;
    }
    s_u[lane] = u; s_ub[lane] = ub;
  }
}

template <int KC, bool SMALL>
__global__ void __launch_bounds__(STREAM_BLOCK, grad_bps<KC>())
nll_grad_kernel(const double2 *__restrict__ a, const double *__restrict__ t, int64_t ld, int64_t n,
                const __grid_constant__ RateParams R, const __grid_constant__ GradParams GP, const double *__restrict__ G,
                double inv_n_norm, double sum_t, double *__restrict__ partials /* [grid][NB * 32 + 5] */, unsigned int *ticket,
                double *__restrict__ result, unsigned long long *stamps /* in-kernel timing while profiling (nll_finish), else NULL */) {
  constexpr int NB = grad_nb<KC>(), XS = gram_stride(NB), NS = 2, NA = NB * 32 + NS;
  if (stamps && threadIdx.x == 0) atomicMin(stamps, global_ns());
  extern __shared__ __align__(16) char smem_raw[];
  __shared__ double s_red[STREAM_WARPS * NA];
  __shared__ double s_sum[NA];
  __shared__ double s_p[STREAM_WARPS];
  __shared__ long long s_e[STREAM_WARPS];
  __shared__ int s_b[STREAM_WARPS];
  __shared__ double s_n[4];
  __shared__ double2 s_u[KC], s_ub[KC];
  __shared__ bool last;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  double *Xs = reinterpret_cast<double *>(smem_raw + (size_t)warp * grad_warp_bytes<KC>());
  double *Wt = Xs + align_up((size_t)32 * XS * sizeof(double), 128) / sizeof(double);
  double *xrow = Xs + lane * XS, *wrow = Wt + lane * GRAD_WS;
#pragma unroll
  for (int c = 0; c < XS; ++c) xrow[c] = 0.0;               // features beyond 2 K_c and the weight rows 4..7 stay zero
#pragma unroll
  for (int c = 0; c < GRAD_WS; ++c) wrow[c] = 0.0;
  MantAcc la;
  double acc[NB][2], sc[NS] = {0.0, 0.0};
#pragma unroll
  for (int b = 0; b < NB; ++b) acc[b][0] = acc[b][1] = 0.0;
  const double yG = R.y * R.Gamma, xG = R.x * R.Gamma;
  const int64_t stride = (int64_t)gridDim.x * STREAM_BLOCK;
  // Whole warps iterate together (the MMA is warp-wide), one tile per iteration.  Measured at K_c = 8, 1 M events (ncu
  // gpu__time_duration, before the two-level grid reduction): this form 38 us; two tiles per iteration (their loads issued
  // together) 40 us; columns brought in by cp.async, double buffered, straight into the X tile 50 us; bulk L2
  // prefetch of the warp's next tile (nine UBLKPF per tile): memory stalls 43 -> 27 % of the warp samples, duration unchanged.  The
  // kernel issues ~440 warp instructions per 32 events, ~300 of them on the fp64 pipe (2 cycles each) plus 16 DMMA: about
  // 16 us of fp64-pipe time per million events on B200's 64 lanes per clock per SM -- it is bound by that pipe and by the
  // serial dependency chain of one event, not by the 136 B per event it streams.
  auto process = [&](const double2 (&v)[KC], double tcur, bool live) {
    double2 A = make_double2(0.0, 0.0), Ab = make_double2(0.0, 0.0);
#pragma unroll
    for (int c = 0; c < KC; ++c) {
      amp_add(A, Ab, R.c[c][0], R.c[c][1], R.cbar[c][0], R.cbar[c][1], v[c]);
      *reinterpret_cast<double2 *>(xrow + 2 * c) = v[c];
    }
    double ch, sh, cs, sn;
    mixing_functions<SMALL>(yG * tcur, xG * tcur, ch, sh, cs, sn);
    const Bilinears q = bilinears(A, Ab);
    const double aa = q.aa, bb = q.bb, cre = q.cre, cim = q.cim;
    const double B = rate_form(q, ch, cs, sh, sn);                                        // the bits of bracket()
    double inv = 0.0;
    if (live) { la.add(B); inv = 1.0 / B; }
    // conj(gA) / B and conj(gAbar) / B as (Re, Im) pairs: the weights of this event
    *reinterpret_cast<double2 *>(wrow) = make_double2(((ch + cs) * A.x - (sh * Ab.x - sn * Ab.y)) * inv, ((ch + cs) * A.y - (sh * Ab.y + sn * Ab.x)) * inv);
    *reinterpret_cast<double2 *>(wrow + 2) = make_double2(((ch - cs) * Ab.x - (sh * A.x + sn * A.y)) * inv, ((ch - cs) * Ab.y - (sh * A.y - sn * A.x)) * inv);
    const double gt = R.Gamma * tcur * inv;
    sc[0] += gt * (-(aa - bb) * sn - 2.0 * cim * cs);
    sc[1] += gt * ((aa + bb) * sh - 2.0 * cre * ch);
    grad_mma_tile<NB>(Xs, Wt, acc);
  };
  auto load_tile = [&](double2 (&v)[KC], double &tt, int64_t first) {
    const int64_t i = first + lane;
    const bool live = i < n;
#pragma unroll
    for (int c = 0; c < KC; ++c) v[c] = live ? ldg_stream2(a + c * ld + i) : make_double2(0.0, 0.0);
    tt = live ? ldg_stream1(t + i) : 0.0;
  };
  constexpr bool TWO = false;                             // two tiles per iteration: measured slower (40 against 38 us)
#pragma unroll 1
  for (int64_t i0 = (int64_t)blockIdx.x * STREAM_BLOCK + warp * 32; i0 < n; i0 += (TWO ? 2 : 1) * stride) {
    double2 va[KC], vb[TWO ? KC : 1];
    double ta, tb = 0.0;
    const bool second = TWO && i0 + stride < n;            // warp-uniform
    load_tile(va, ta, i0);
    if (TWO) {
      if (second) load_tile(reinterpret_cast<double2 (&)[KC]>(vb), tb, i0 + stride);
    }
    process(va, ta, i0 + lane < n);
    if (TWO) {
      if (second) process(reinterpret_cast<const double2 (&)[KC]>(vb), tb, i0 + stride + lane < n);
    }
  }
  const bool fin = grad_reduce<NB, NS>(acc, sc, la, partials, ticket, s_red, s_sum, s_p, s_e, s_b, &last);
  if (!fin) return;
  if (warp == 1) {
    double nAA, nBB, xr, xi;
    gram_sums_warp(R, G, KC, inv_n_norm, nAA, nBB, xr, xi);
    if (lane == 0) { s_n[0] = nAA; s_n[1] = nBB; s_n[2] = xr; s_n[3] = xi; }
  } else if (warp == 2) {
    grad_gram_vectors<KC>(R, G, inv_n_norm, lane, s_u, s_ub);
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
    // Re D_k = sum (gx vx + gy vy), Im D_k = sum (gx vy - gy vx); W rows: 0 gx, 1 gy, 2 hx, 3 hy; features 2k (Re), 2k+1 (Im)
    const double dre = grad_c(s_sum, 0, 2 * tid) + grad_c(s_sum, 1, 2 * tid + 1), dim = grad_c(s_sum, 0, 2 * tid + 1) - grad_c(s_sum, 1, 2 * tid);
    const double ere = grad_c(s_sum, 2, 2 * tid) + grad_c(s_sum, 3, 2 * tid + 1), eim = grad_c(s_sum, 2, 2 * tid + 1) - grad_c(s_sum, 3, 2 * tid);
    double *g = result + GRAD_OFFSET;
    g[2 * tid] = -2.0 * dre + scale * 2.0 * hr;
    g[2 * tid + 1] = 2.0 * dim + scale * 2.0 * hi;
    g[2 * KC + 2 * tid] = -2.0 * ere + scale * 2.0 * br;
    g[2 * KC + 2 * tid + 1] = 2.0 * eim + scale * 2.0 * bi;
  }
  if (tid == 0) {
    double *g = result + GRAD_OFFSET;
    g[4 * KC] = -s_sum[NB * 32] + scale * (GP.dT1dx * (nAA - nBB) - 2.0 * GP.dT3dx * xi);
    g[4 * KC + 1] = -s_sum[NB * 32 + 1] + scale * (GP.dT0dy * (nAA + nBB) - 2.0 * GP.dT2dy * xr);
    const double prod = s_p[0];
    const long long esum = s_e[0];
    const int bad = s_b[0];
    double s0 = log(prod) + 0.693147180559945309417 * (double)esum;
    double nll = R.Gamma * sum_t - s0 + (double)n * log(norm);
    if (bad > 0 || !(norm > 0.0)) nll = INFINITY;
    result[0] = s0; result[1] = sum_t; result[2] = norm; result[3] = nll; result[4] = (double)bad;
    *ticket = 0;
    if (stamps) {
      const unsigned long long t1 = global_ns(), t0 = *reinterpret_cast<volatile unsigned long long *>(stamps);
      atomicAdd(stamps + 1, t1 - t0);
      atomicAdd(stamps + 2, 1ull);
      *reinterpret_cast<volatile unsigned long long *>(stamps) = ~0ull;
    }
  }
}

// ------------------------------------------------------------------------------------------------
// The same in resolution mode (config 5): P_i = R_i / N_i with R_i the bracket with the convolved time functions psi_m of
// the event and N_i = sum_m T_m(sigma_i) S_m (stream_kernels.cuh, resolved_prob).  Per event the kernel reads the K_c
// columns, the eight time rows and the eight derivative rows (tres_grad_kernel).  d(sum log N_i)/dc_k* keeps the Gram
// structure with per-call weights W_m = sum_i T_m,i / N_i:  (W0+W1) u_k - (W2 + i W3) ubar_k.
template <int KC>
__global__ void __launch_bounds__(STREAM_BLOCK, STREAM_BLOCKS_PER_SM)
nll_grad_res_kernel(const double2 *__restrict__ a, const double *__restrict__ tr, const double *__restrict__ trg, int64_t ld,
                    int64_t n, const __grid_constant__ RateParams R, const double *__restrict__ G, double inv_n_norm,
                    double *__restrict__ partials /* [grid][NB * 32 + 9] */, unsigned int *ticket, double *__restrict__ result) {
  constexpr int NB = grad_nb<KC>(), XS = gram_stride(NB), NS = 6, NC = NB * 32, NA = NC + NS;
  extern __shared__ __align__(16) char smem_raw[];
  __shared__ double s_red[STREAM_WARPS * NA];
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
  double *Xs = reinterpret_cast<double *>(smem_raw + (size_t)warp * grad_warp_bytes<KC>());
  double *Wt = Xs + align_up((size_t)32 * XS * sizeof(double), 128) / sizeof(double);
  double *xrow = Xs + lane * XS, *wrow = Wt + lane * GRAD_WS;
#pragma unroll
  for (int c = 0; c < XS; ++c) xrow[c] = 0.0;
#pragma unroll
  for (int c = 0; c < GRAD_WS; ++c) wrow[c] = 0.0;
  MantAcc la;
  double acc[NB][2], sc[NS];
#pragma unroll
  for (int b = 0; b < NB; ++b) acc[b][0] = acc[b][1] = 0.0;
#pragma unroll
  for (int j = 0; j < NS; ++j) sc[j] = 0.0;
  const int64_t stride = (int64_t)gridDim.x * STREAM_BLOCK;
#pragma unroll 1
  for (int64_t i0 = (int64_t)blockIdx.x * STREAM_BLOCK + warp * 32; i0 < n; i0 += stride) {
    const int64_t i = i0 + lane;
    const bool live = i < n;
    double2 v[KC];
    double w[8], d[8];
#pragma unroll
    for (int c = 0; c < KC; ++c) v[c] = live ? ldg_stream2(a + c * ld + i) : make_double2(0.0, 0.0);
#pragma unroll
    for (int m = 0; m < 8; ++m) { w[m] = live ? ldg_stream1(tr + m * ld + i) : 1.0; d[m] = live ? ldg_stream1(trg + m * ld + i) : 0.0; }
    double2 A = make_double2(0.0, 0.0), Ab = make_double2(0.0, 0.0);
#pragma unroll
    for (int c = 0; c < KC; ++c) {
      amp_add(A, Ab, R.c[c][0], R.c[c][1], R.cbar[c][0], R.cbar[c][1], v[c]);
      *reinterpret_cast<double2 *>(xrow + 2 * c) = v[c];
    }
    const Bilinears q = bilinears(A, Ab);
    const double aa = q.aa, bb = q.bb, cre = q.cre, cim = q.cim;
    const double Rv = rate_form(q, w[0], w[1], w[2], w[3]);                                        // the bits of resolved_prob()
    const double Nv = fma(S1, w[4], fma(S2, w[5], fma(-2.0 * S3, w[6], __dmul_rn(-2.0 * S4, w[7]))));
    double invR = 0.0, invN = 0.0;
    if (live) { la.add(__ddiv_rn(Rv, Nv)); invR = 1.0 / Rv; invN = 1.0 / Nv; }
    *reinterpret_cast<double2 *>(wrow) = make_double2(((w[0] + w[1]) * A.x - (w[2] * Ab.x - w[3] * Ab.y)) * invR, ((w[0] + w[1]) * A.y - (w[2] * Ab.y + w[3] * Ab.x)) * invR);
    *reinterpret_cast<double2 *>(wrow + 2) = make_double2(((w[0] - w[1]) * Ab.x - (w[2] * A.x + w[3] * A.y)) * invR, ((w[0] - w[1]) * Ab.y - (w[2] * A.y - w[3] * A.x)) * invR);
    // d log(R/N) / dx, / dy: d = (dpsi1/dx, dpsi3/dx, dpsi0/dy, dpsi2/dy, dT1/dx, dT3/dx, dT0/dy, dT2/dy)
    sc[0] += ((aa - bb) * d[0] - 2.0 * cim * d[1]) * invR - (S2 * d[4] - 2.0 * S4 * d[5]) * invN;
    sc[1] += ((aa + bb) * d[2] - 2.0 * cre * d[3]) * invR - (S1 * d[6] - 2.0 * S3 * d[7]) * invN;
#pragma unroll
    for (int m = 0; m < 4; ++m) sc[2 + m] = fma(w[4 + m], invN, sc[2 + m]);     // W_m
    grad_mma_tile<NB>(Xs, Wt, acc);
  }
  const bool fin = grad_reduce<NB, NS>(acc, sc, la, partials, ticket, s_red, s_sum, s_p, s_e, s_b, &last);
  if (!fin) return;
  if (warp == 2) grad_gram_vectors<KC>(R, G, inv_n_norm, lane, s_u, s_ub);
  __syncthreads();
  const double W0 = s_sum[NC + 2], W1 = s_sum[NC + 3], W2 = s_sum[NC + 4], W3 = s_sum[NC + 5];
  double *g = result + GRAD_OFFSET;
  if (tid < KC) {
    const double2 u = s_u[tid], ub = s_ub[tid];
    const double hr = (W0 + W1) * u.x - (W2 * ub.x - W3 * ub.y), hi = (W0 + W1) * u.y - (W2 * ub.y + W3 * ub.x);
    const double br = (W0 - W1) * ub.x - (W2 * u.x + W3 * u.y), bi = (W0 - W1) * ub.y - (W2 * u.y - W3 * u.x);
    const double dre = grad_c(s_sum, 0, 2 * tid) + grad_c(s_sum, 1, 2 * tid + 1), dim = grad_c(s_sum, 0, 2 * tid + 1) - grad_c(s_sum, 1, 2 * tid);
    const double ere = grad_c(s_sum, 2, 2 * tid) + grad_c(s_sum, 3, 2 * tid + 1), eim = grad_c(s_sum, 2, 2 * tid + 1) - grad_c(s_sum, 3, 2 * tid);
    g[2 * tid] = -2.0 * dre + 2.0 * hr;
    g[2 * tid + 1] = 2.0 * dim + 2.0 * hi;
    g[2 * KC + 2 * tid] = -2.0 * ere + 2.0 * br;
    g[2 * KC + 2 * tid + 1] = 2.0 * eim + 2.0 * bi;
  }
  if (tid == 0) {
    g[4 * KC] = -s_sum[NC];
    g[4 * KC + 1] = -s_sum[NC + 1];
    const double s0 = log(s_p[0]) + 0.693147180559945309417 * (double)s_e[0];
    const double norm = R.T[0] * S1 + R.T[1] * S2 - 2.0 * R.T[2] * S3 - 2.0 * R.T[3] * S4;
    double nll = -s0;
    if (s_b[0] > 0 || !(norm > 0.0)) nll = INFINITY;
    result[0] = s0; result[1] = 0.0; result[2] = norm; result[3] = nll; result[4] = (double)s_b[0];
    *ticket = 0;
  }
}

}  // namespace tddp4k
