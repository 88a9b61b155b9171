// colnll_jit.cuh -- the data pass after a mass or width moved: lineshapes of the
// changed model (O-6), coupling columns a_kappa = sum_{k in kappa} f_k T_R1(k) T_R2(k) (eq. (2)),
// the rate of eq. (1) and the -sum log reduction, in one pass over the static cache of the data sample.  Reads the s rows
// in use, the g rows, the f rows and t (resolution mode: the eight time rows); writes the stale coupling columns back for
// the coupling-only calls that follow and finishes the NLL in the same pass.
//
// NOT compiled by nvcc: the library compiles this file at run time with NVRTC (jit.h), once per model, behind the same
// generated prelude as gram_jit.cuh (model tables as compile-time constants) plus
//   J_SMALL  1: |x Gamma t|, |y Gamma t| < 1/4 over the sample, Taylor forms of the four time functions,
//   J_RES    1: per-event resolution (config 5) or time-integrated mode: t points at the time rows [8][ld].
// Lineshapes stay in registers, every table entry is an immediate (see gram_jit.cuh for the measurements behind this).
// Same grid, same event-to-thread map, same per-event arithmetic (nll_shared.cuh) as nll_stream_kernel: a rebuilt call
// returns the bits a cached call returns.
#include "nll_shared.cuh"

namespace tddp4k {

extern "C" __global__ void __launch_bounds__(STREAM_BLOCK, STREAM_BLOCKS_PER_SM)
colnll_jit(const __grid_constant__ LineParams LP, const double *__restrict__ cache, const double *__restrict__ t,
           long long ld, long long n, double2 *__restrict__ a, const __grid_constant__ RateParams R,
           const double *__restrict__ G, double inv_n_norm, double sum_t, double *__restrict__ partials, unsigned int *ticket,
           double *__restrict__ result, int early_wait,
           unsigned int store_mask /* bit kappa: the stored column kappa is stale and is rewritten */, double seq) {
  constexpr bool SMALL = J_SMALL != 0, RES = J_RES != 0;
  __shared__ double s_S[4];
  if (RES || early_wait) pdl_wait();       // the predecessor reads the columns this kernel rewrites (or RES: G first)
  pdl_launch_dependents();
  const int lane = threadIdx.x & 31;
  MantAcc la;
  const double yG = R.y * R.Gamma, xG = R.x * R.Gamma;
  const long long stride = (long long)gridDim.x * STREAM_BLOCK;
  if (RES) block_phase_space_sums(R, G, J_KC, inv_n_norm, s_S);
  long long i = (long long)blockIdx.x * STREAM_BLOCK + threadIdx.x;
#pragma unroll 1
  for (; i < n; i += stride) {
    if (PF_DIST > 0 && J_R * 32 - J_SKIP > 0 && lane == 0 && i + PF_DIST * stride < n)
      prefetch_l2_bulk(tile_event(cache, J_R, i + PF_DIST * stride) + J_SKIP, (unsigned)(J_R * 32 - J_SKIP) * 8u);
    const double ti = RES ? 0.0 : ldg_stream1(t + i);            // RES: t points at the time rows [8][ld]
    const double *ev = tile_event(cache, J_R, i);
    double sv[J_NSU + 2], gv[J_NG + 1], fv[J_NF + 1];               // + 1: a model without resonances has no instance
#pragma unroll
    for (int r = 0; r < J_NSU; ++r) sv[r] = ldg_stream1(ev + J_SKIP + r * 32);
#pragma unroll
    for (int r = 0; r < J_NG; ++r) gv[r] = ldg_stream1(ev + J_GOFF + r * 32);
#pragma unroll
    for (int r = 0; r < J_NF; ++r) fv[r] = ldg_stream1(ev + J_FOFF + r * 32);
#if J_NSD
    {                                                      // the s that is not streamed: a fixed combination of streamed rows
      double d = J_SDCONST;
#pragma unroll
      for (int r = 0; r < J_NSU; ++r)
        if (J_SDCOEF[r] > 0) d += sv[r];
        else if (J_SDCOEF[r] < 0) d -= sv[r];
      sv[J_NSU] = d;
    }
#endif
    double2 T[J_NINST + 1];
#pragma unroll
    for (int j = 0; j < J_NINST; ++j) T[j] = breit_wigner(LP.m0sq[j], LP.gam[j], sv[J_SROW[j]], gv[J_GROW[j]]);
    double2 A = make_double2(0.0, 0.0), Ab = make_double2(0.0, 0.0);
    double2 col = make_double2(0.0, 0.0);
#pragma unroll
    for (int k = 0; k < J_NTERMS; ++k) {
      double2 P;
      if (J_T0[k] >= 0 && J_T1[k] >= 0) P = cmul(T[J_T0[k] >= 0 ? J_T0[k] : 0], T[J_T1[k] >= 0 ? J_T1[k] : 0]);
      else if (J_T0[k] >= 0) P = T[J_T0[k] >= 0 ? J_T0[k] : 0];
      else if (J_T1[k] >= 0) P = T[J_T1[k] >= 0 ? J_T1[k] : 0];
      else P = make_double2(1.0, 0.0);
      const double fk = J_FROW[k] >= 0 ? fv[J_FROW[k] >= 0 ? J_FROW[k] : 0] : 1.0;    // non-resonant term: no row, f = 1
      col.x = fma(fk, P.x, col.x);
      col.y = fma(fk, P.y, col.y);
      if (J_LAST[k]) {
        // a column none of whose lineshapes moved is recomputed to the bits already stored: skip its 16-byte store
        if ((store_mask >> J_COL[k]) & 1u) a[(long long)J_COL[k] * ld + i] = col;
        amp_add(A, Ab, R.c[J_COL[k]][0], R.c[J_COL[k]][1], R.cbar[J_COL[k]][0], R.cbar[J_COL[k]][1], col);
        col = make_double2(0.0, 0.0);
      }
    }
    if (RES) la.add(resolved_prob(A, Ab, t + i, ld, s_S));
    else la.add(bracket<SMALL>(A, Ab, yG * ti, xG * ti));
  }
  if (!(RES || early_wait)) pdl_wait();
  nll_finish<RES>(R, J_KC, n, sum_t, la, G, inv_n_norm, partials, ticket, result, seq);
}

}  // namespace tddp4k
