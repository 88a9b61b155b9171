// gram_jit.cuh -- step 6 (the normalisation "from several million phase space
// points"), fused with steps 2+3 over the static cache of the normalisation sample:
//     G_kl = sum_j w_j a_k(p_j) conj(a_l(p_j))        (K_c x K_c Hermitian; O-8: N is a contraction of G with the couplings)
// The columns of the normalisation sample are never stored.  With x_j = (Re a_0, Im a_0, Re a_1, ...) the real matrix
// X^T diag(w) X holds every Re/Im piece of G, and it is a dense contraction over events: it runs on the fp64 tensor cores
// (mma.sync m8n8k4, SASS DMMA), the only place of the path where they apply (north_star):
//   G_kl.re = XtX[2k][2l] + XtX[2k+1][2l+1],   G_kl.im = XtX[2k+1][2l] - XtX[2k][2l+1].
//
// This file is NOT compiled by nvcc.  The library compiles it at run time with NVRTC (jit.h), once per model, behind a
// generated prelude that states the model as compile-time constants:
//   J_NB, J_KC, J_NINST, J_NTERMS, J_NSU, J_NG, J_NF (s, g, f rows streamed), J_R, J_SKIP, J_GOFF, J_FOFF, J_WOFF (element
//   offsets in a tile, -1: unweighted), J_GROW[J_NINST], J_FROW[J_NTERMS]  the (shared) g row of instance j / f row of term k,
//   J_SROW[J_NINST]  index (0 .. J_NSU-1) of the s row instance j reads, rows counted from J_SKIP,
//   J_T0[J_NTERMS], J_T1[J_NTERMS]  lineshape instances of term k (-1: none),  J_COL[J_NTERMS]  its coupling column,
//   J_LAST[J_NTERMS]  1: term k closes its column (terms are sorted by column).
// Why: PAPER.md line 51 builds the amplitude from tables of shared lineshape / spin-factor instances.  A table-driven
// kernel has to park the lineshapes T_R of an event in shared memory, because the terms index them at run time: per
// 32-event tile that was 13 STS.128 + 32 LDS.128 of lineshapes next to the loads themselves, the X tile and the MMA
// fragments -- 342 wavefronts of the LSU data pipe per tile, and ncu showed that pipe 80-82 % busy with no other unit
// above 45 %: the kernel sat at 0.82-0.85 of the HBM roofline on the shared-memory pipe, not on bytes.  With the tables
// compile-time constants every index below is an immediate: the lineshapes stay in registers (no scratch at all), every
// load carries an immediate offset, and the per-term table lookups, address arithmetic and flush branches disappear.
// Deterministic: per-warp accumulation in event order, warps, blocks and block groups summed in index order.
//
// J_GMODE (the incremental update of G; tddp4_set_gram_mode):
//   0  plain pass: nothing of the normalisation sample is stored (the default);
//   1  full pass that also stores the coupling columns whose bit is set in `mask` into an[K_c][ld];
//   2  incremental pass: columns whose bit is clear in `mask` are READ from an (16 B), only the masked ones are rebuilt
//      from the rows of their terms (J_INSTCOLS / J_SROWCOLS: the columns each lineshape instance / s row feeds) and
//      written back.  Same tiles, same arithmetic, same accumulation order: G has the bits of a full pass.
#include "jit_shared.cuh"

namespace tddp4k {

constexpr int JG_BLOCK = 256;

extern "C" __global__ void __launch_bounds__(JG_BLOCK, J_BPS)
gram_jit(const __grid_constant__ LineParams LP, const double *__restrict__ cache, long long n,
         double *__restrict__ partials /* [grid + groups][64 NB NB] */, unsigned int *ticket,
         double *__restrict__ G /* [KC][KC][2] sums, Hermitian, full */,
         double2 *__restrict__ an /* J_GMODE > 0: stored columns [KC][ld] */, long long ld, unsigned int mask) {
  constexpr int GMODE = J_GMODE;
  constexpr int NB = J_NB, F = 8 * NB, STRIDE = gram_stride(NB), NP = NB * (NB + 1) / 2;
  constexpr bool WEIGHTED = J_WOFF >= 0;
  extern __shared__ __align__(16) char smem_raw[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  double *Xs = reinterpret_cast<double *>(smem_raw) + (size_t)warp * 32 * STRIDE;   // [32][STRIDE]: row = event
  double *row = Xs + lane * STRIDE;
#pragma unroll
  for (int c = 0; c < STRIDE; ++c) row[c] = 0.0;                // features beyond 2 K_c stay zero
  double acc[NP][2];
#pragma unroll
  for (int q = 0; q < NP; ++q) acc[q][0] = acc[q][1] = 0.0;
  const long long stride = (long long)gridDim.x * JG_BLOCK;
  // whole warps iterate together (the MMA is warp-wide).  The cache is allocated and zero-filled in whole tiles, so the
  // lanes of a ragged last tile compute on zeros: f = 0 gives zero columns, and their weight is forced to 0.
  long long i0 = (long long)blockIdx.x * JG_BLOCK + warp * 32;
#pragma unroll 1
  for (; i0 < n; i0 += stride) {
    if (GMODE != 2 && PF_DIST > 0 && J_R * 32 - J_SKIP > 0 && lane == 0 && i0 + PF_DIST * stride < n)     // (an incremental pass reads part of a tile only)
      prefetch_l2_bulk(tile_event(cache, J_R, i0 + PF_DIST * stride) + J_SKIP, (unsigned)(J_R * 32 - J_SKIP) * 8u);
    const double *ev = tile_event(cache, J_R, i0 + lane);
    double sv[J_NSU + 2], gv[J_NG + 1], fv[J_NF + 1];          // + 1: a model without resonances has no instance
    double2 kept[J_KC];                                    // GMODE 2: the clean columns, read back
    if (GMODE == 2) {                                      // only the rows the masked columns need (warp-uniform guards)
#pragma unroll
      for (int c = 0; c < J_KC; ++c) kept[c] = (mask >> c) & 1u ? make_double2(0.0, 0.0) : ldg_stream2(an + c * ld + i0 + lane);
#pragma unroll
      for (int r = 0; r < J_NSU; ++r) sv[r] = (mask & J_SROWCOLS[r]) ? ldg_stream1(ev + J_SKIP + r * 32) : 0.0;
#pragma unroll
      for (int r = 0; r < J_NG; ++r) gv[r] = (mask & J_GROWCOLS[r]) ? ldg_stream1(ev + J_GOFF + r * 32) : 0.0;
#pragma unroll
      for (int r = 0; r < J_NF; ++r) fv[r] = (mask & J_FROWCOLS[r]) ? ldg_stream1(ev + J_FOFF + r * 32) : 0.0;
    } else {
#pragma unroll
      for (int r = 0; r < J_NSU; ++r) sv[r] = ldg_stream1(ev + J_SKIP + r * 32);
#pragma unroll
      for (int r = 0; r < J_NG; ++r) gv[r] = ldg_stream1(ev + J_GOFF + r * 32);
#pragma unroll
      for (int r = 0; r < J_NF; ++r) fv[r] = ldg_stream1(ev + J_FOFF + r * 32);
    }
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
    double wj = 1.0;
    if (WEIGHTED) wj = ldg_stream1(ev + J_WOFF);
    double2 T[J_NINST + 1];
#pragma unroll
    for (int j = 0; j < J_NINST; ++j)
      if (GMODE != 2 || (mask & J_INSTCOLS[j])) T[j] = breit_wigner(LP.m0sq[j], LP.gam[j], sv[J_SROW[j]], gv[J_GROW[j]]);
      else T[j] = make_double2(0.0, 0.0);
    double2 a = make_double2(0.0, 0.0);
    const double one = i0 + lane < n ? 1.0 : 0.0;          // lanes beyond n: rows are zero-filled, the constant f must be too
#pragma unroll
    for (int k = 0; k < J_NTERMS; ++k) {
      double2 P;
      if (J_T0[k] >= 0 && J_T1[k] >= 0) P = cmul(T[J_T0[k] >= 0 ? J_T0[k] : 0], T[J_T1[k] >= 0 ? J_T1[k] : 0]);
      else if (J_T0[k] >= 0) P = T[J_T0[k] >= 0 ? J_T0[k] : 0];
      else if (J_T1[k] >= 0) P = T[J_T1[k] >= 0 ? J_T1[k] : 0];
      else P = make_double2(1.0, 0.0);
      const double fk = J_FROW[k] >= 0 ? fv[J_FROW[k] >= 0 ? J_FROW[k] : 0] : one;    // non-resonant term: no row, f = 1
      a.x = fma(fk, P.x, a.x);
      a.y = fma(fk, P.y, a.y);
      if (J_LAST[k]) {
        if (GMODE == 2 && !((mask >> J_COL[k]) & 1u)) a = kept[J_COL[k]];
        if (GMODE != 0 && ((mask >> J_COL[k]) & 1u)) an[J_COL[k] * ld + i0 + lane] = a;
        *reinterpret_cast<double2 *>(row + 2 * J_COL[k]) = a;
        a = make_double2(0.0, 0.0);
      }
    }
    if (WEIGHTED) row[F] = i0 + lane < n ? wj : 0.0;
    __syncwarp();
    {
      const double *base = Xs + (2 * (lane & 3)) * STRIDE + (lane >> 2);
#pragma unroll
      for (int grp = 0; grp < 8; ++grp) {                  // 4 events per MMA, 8 groups per warp tile
        const double *r = base + (8 * (grp >> 1) + (grp & 1)) * STRIDE;
        double x[NB];
#pragma unroll
        for (int b = 0; b < NB; ++b) x[b] = r[8 * b];
        double wv = 1.0;
        if (WEIGHTED) wv = r[F - (lane >> 2)];
        int q = 0;
#pragma unroll
        for (int bi = 0; bi < NB; ++bi) {
          const double aw = WEIGHTED ? wv * x[bi] : x[bi];
#pragma unroll
          for (int bj = bi; bj < NB; ++bj, ++q) dmma884(acc[q][0], acc[q][1], aw, x[bj]);
        }
      }
    }
    __syncwarp();                                          // the X tile is free again
  }
  __syncthreads();                                         // the X tiles are free: the reduction reuses the memory
  gram_reduce_tail<NB, JG_BLOCK>(acc, reinterpret_cast<double *>(smem_raw), J_KC, partials, ticket, G);
}

}  // namespace tddp4k
