// stream_kernels.cuh -- the three per-call kernels of the NLL path, all on the TMA tile pipeline of tile_pipe.cuh:
//   nll_stream_kernel     steps 4+5+7   over cached coupling columns            (coupling / x / y / tau-only call)
//   colnll_stream_kernel  steps 2..5+7  over the step-1 caches of the data set  (call after a mass or width moved)
//   gram_stream_kernel    steps 2+3+6   over the step-1 caches of the normalisation set (fp64 tensor-core Gram)
// All use TILE threads per block, one event per thread per tile, persistent blocks (grid = min(tiles, #SM)).  Because
// nll_stream and colnll_stream give every event to the same thread in the same order, the fixed-order reduction
// returns bit-identical NLLs whether the columns were cached or rebuilt in the call.
#pragma once
#include "tile_pipe.cuh"

namespace tddp4k {

// shared-memory carve-up helpers -------------------------------------------------------------------------------
__host__ __device__ constexpr size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// Lineshapes + component products of ONE event from a staged tile (steps 2+3).  The stage starts with the s rows in
// use, then the g rows (one per instance), then the f rows (one per term), all doubles.  T_R of every instance goes
// to the warp's private scratch sT[instance][lane]; chains index it through the model tables (P:51 de-duplication).
template <int KCMAX, int TILE>
__device__ __forceinline__ void staged_columns(const ModelTab &M, const LineParams &LP, const double *st, int tid,
                                               double2 *sT /* warp-private [n_inst][32] */, int lane,
                                               double2 col[KCMAX]) {
  const double *gs = st + M.n_su * TILE, *fs = gs + M.n_inst * TILE;
  for (int j = 0; j < M.n_inst; ++j)
    sT[j * 32 + lane] = breit_wigner(LP.m0sq[j], LP.gam[j], st[M.sys_slot[M.inst[j].sys] * TILE + tid], gs[j * TILE + tid]);
#pragma unroll
  for (int kap = 0; kap < KCMAX; ++kap) {
    double2 acc = make_double2(0.0, 0.0);
    for (int k = M.col_begin[kap]; k < M.col_begin[kap + 1]; ++k) {      // empty beyond K_c (col_begin is 0 there)
      const TermTab &tm = M.term[k];
      double fv = fs[k * TILE + tid];
      double2 T = make_double2(1.0, 0.0);
      if (tm.inst0 >= 0) T = cmul(sT[tm.inst0 * 32 + lane], sT[tm.inst1 * 32 + lane]);
      acc.x += fv * T.x;
      acc.y += fv * T.y;
    }
    col[kap] = acc;
  }
}

// ------------------------------------------------------------------------------------------------
// Coupling-only call.  Rows: K_c columns (16 B elements), then t.  Algorithmic traffic 16 K_c + 8 B per event.
template <int TILE>
__host__ __device__ constexpr int nll_stages() { return TILE == 256 ? 4 : 8; }
template <int TILE>
inline size_t nll_smem_bytes(int KC) { return 128 + (size_t)nll_stages<TILE>() * TILE * (16 * KC + 8); }

template <int KC, bool PROB, bool SMALL, int TILE>
__global__ void __launch_bounds__(TILE, 1)
nll_stream_kernel(const __grid_constant__ RowList rows, int64_t ld, int64_t n, const __grid_constant__ RateParams R,
                  const double *__restrict__ G, double inv_n_norm, double sum_t, double *__restrict__ partials,
                  unsigned int *ticket, double *__restrict__ result, double *__restrict__ prob_out) {
  constexpr int STAGES = nll_stages<TILE>();
  extern __shared__ __align__(128) char smem_raw[];
  char *smem = smem_raw;
  __shared__ double red[TILE / 32];
  __shared__ double s_norm;
  __shared__ bool last;
  TilePipe<TILE, STAGES> pipe(reinterpret_cast<uint64_t *>(smem), smem + 128, rows, n, ld);
  pipe.init();
  pipe.prologue();
  double norm0 = 0.0;
  if (PROB || blockIdx.x == 0) {                         // block 0 evaluates N while its first tiles are in flight
    norm0 = norm_from_gram<TILE>(R, G, KC, inv_n_norm, red);
    if (PROB) {
      if (threadIdx.x == 0) s_norm = norm0;
      __syncthreads();
    }
  }
  LogAcc la;
  const double yG = R.y * R.Gamma, xG = R.x * R.Gamma;
  const int tid = threadIdx.x;
  int64_t k = 0;
  for (int64_t tile = blockIdx.x; tile < pipe.n_tiles; tile += gridDim.x, ++k) {
    const char *st = pipe.wait(k);
    int64_t i = tile * TILE + tid;
    if (i < n) {
      double2 v[KC];
#pragma unroll
      for (int c = 0; c < KC; ++c) v[c] = reinterpret_cast<const double2 *>(st + (size_t)c * TILE * 16)[tid];
      double ti = reinterpret_cast<const double *>(st + (size_t)KC * TILE * 16)[tid];
      double2 A, Ab;
      amplitude_sums<KC>(R, v, A, Ab);
      double B = bracket<SMALL>(A, Ab, yG * ti, xG * ti);
      la.add(B);
      if (PROB) prob_out[i] = exp(-R.Gamma * ti) * B / s_norm;
    }
    __syncthreads();                                     // every thread is done with this stage
    pipe.refill(k);
  }
  nll_finish<TILE>(R, n, sum_t, la.value(), (double)la.bad, norm0, partials, ticket, result, red, &last);
}

// ------------------------------------------------------------------------------------------------
// Call after a mass or width moved, data set.  Rows: s rows in use, g rows, f rows, then t.  Writes every coupling
// column back (for the coupling-only calls that follow) and finishes the NLL in the same pass.
template <int TILE>
inline size_t colnll_smem_bytes(int bytes_per_event, int n_inst) {
  return 128 + (size_t)2 * TILE * bytes_per_event + (size_t)(TILE / 32) * (n_inst > 0 ? n_inst : 1) * 32 * sizeof(double2);
}

template <int KC, bool SMALL, int TILE>
__global__ void __launch_bounds__(TILE, 1)
colnll_stream_kernel(const __grid_constant__ ModelTab M, const __grid_constant__ LineParams LP,
                     const __grid_constant__ RowList rows, int64_t ld, int64_t n, double2 *__restrict__ a,
                     const __grid_constant__ RateParams R, const double *__restrict__ G, double inv_n_norm, double sum_t,
                     double *__restrict__ partials, unsigned int *ticket, double *__restrict__ result) {
  constexpr int STAGES = 2;
  extern __shared__ __align__(128) char smem_raw[];
  char *smem = smem_raw;
  __shared__ double red[TILE / 32];
  __shared__ bool last;
  TilePipe<TILE, STAGES> pipe(reinterpret_cast<uint64_t *>(smem), smem + 128, rows, n, ld);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  double2 *sT = reinterpret_cast<double2 *>(smem + 128 + (size_t)STAGES * TILE * rows.bytes_per_event) +
                (size_t)warp * (M.n_inst > 0 ? M.n_inst : 1) * 32;
  pipe.init();
  pipe.prologue();
  double norm0 = 0.0;
  if (blockIdx.x == 0) norm0 = norm_from_gram<TILE>(R, G, KC, inv_n_norm, red);
  LogAcc la;
  const double yG = R.y * R.Gamma, xG = R.x * R.Gamma;
  const int t_slot = M.n_su + M.n_inst + M.n_terms;
  int64_t k = 0;
  for (int64_t tile = blockIdx.x; tile < pipe.n_tiles; tile += gridDim.x, ++k) {
    const double *st = reinterpret_cast<const double *>(pipe.wait(k));
    int64_t i = tile * TILE + tid;
    if (i < n) {
      double2 v[KC];
      staged_columns<KC, TILE>(M, LP, st, tid, sT, lane, v);
      double ti = st[t_slot * TILE + tid];
#pragma unroll
      for (int c = 0; c < KC; ++c) __stcs(a + c * ld + i, v[c]);
      double2 A, Ab;
      amplitude_sums<KC>(R, v, A, Ab);
      la.add(bracket<SMALL>(A, Ab, yG * ti, xG * ti));
    }
    __syncthreads();
    pipe.refill(k);
  }
  nll_finish<TILE>(R, n, sum_t, la.value(), (double)la.bad, norm0, partials, ticket, result, red, &last);
}

// ------------------------------------------------------------------------------------------------
// step 6: Hermitian Gram matrix G_kl = sum_j w_j a_k(p_j) conj(a_l(p_j)) over the normalisation sample, fused with
// steps 2+3: the columns of the normalisation sample are never stored.  With x_j = (Re a_0, Im a_0, Re a_1, ...)
// the real matrix X^T diag(w) X holds every Re/Im piece of G, and it is a dense contraction over events: it runs on
// the fp64 tensor cores (mma.sync m8n8k4, SASS DMMA), the only place of the path where they apply (north_star).
//   G_kl.re = XtX[2k][2l] + XtX[2k+1][2l+1],   G_kl.im = XtX[2k+1][2l] - XtX[2k][2l+1].
// One thread per event computes the columns; each warp then feeds its own 32 events, 4 at a time, through the
// MMA from a padded warp-private tile that re-uses the lineshape scratch.  NB = number of 8-feature blocks.
// Rows: s rows in use, g rows, f rows, then w if the sample is weighted.
// Deterministic: per-warp accumulation in event order, warps then blocks summed in index order.
__host__ __device__ constexpr int gram_stride(int NB) { return NB <= 2 ? 20 : 36; }   // = 4 mod 16: conflict-free fragments
__host__ __device__ inline size_t gram_warp_scratch(int NB, int n_inst) {
  size_t a = (size_t)(n_inst > 0 ? n_inst : 1) * 32 * sizeof(double2), b = (size_t)32 * gram_stride(NB) * sizeof(double);
  return align_up(a > b ? a : b, 128);
}
template <int TILE>
inline size_t gram_smem_bytes(int NB, int bytes_per_event, int n_inst) {
  size_t stages = (size_t)2 * TILE * bytes_per_event, red = (size_t)(TILE / 32) * NB * NB * 64 * sizeof(double);
  return 128 + (stages > red ? stages : red) + (size_t)(TILE / 32) * gram_warp_scratch(NB, n_inst);
}

__device__ __forceinline__ void dmma884(double &c0, double &c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

template <int NB, int TILE>
__global__ void __launch_bounds__(TILE, 1)
gram_stream_kernel(const __grid_constant__ ModelTab M, const __grid_constant__ LineParams LP,
                   const __grid_constant__ RowList rows, int64_t ld, int64_t n, int weighted,
                   double *__restrict__ partials /* [grid][64 NB NB] */, unsigned int *ticket,
                   double *__restrict__ G /* [KC][KC][2] sums, Hermitian, full */) {
  constexpr int STAGES = 2, KCMAX = 4 * NB, F = 8 * NB, STRIDE = gram_stride(NB), NP = NB * (NB + 1) / 2, WARPS = TILE / 32;
  extern __shared__ __align__(128) char smem_raw[];
  char *smem = smem_raw;
  __shared__ bool last;
  TilePipe<TILE, STAGES> pipe(reinterpret_cast<uint64_t *>(smem), smem + 128, rows, n, ld);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int KC = M.n_kc;
  size_t stage_bytes = (size_t)STAGES * TILE * rows.bytes_per_event, red_bytes = (size_t)WARPS * NB * NB * 64 * sizeof(double);
  char *scratch = smem + 128 + (stage_bytes > red_bytes ? stage_bytes : red_bytes) + (size_t)warp * gram_warp_scratch(NB, M.n_inst);
  double2 *sT = reinterpret_cast<double2 *>(scratch);    // [n_inst][32] while the columns are formed ...
  double *Xs = reinterpret_cast<double *>(scratch);      // ... then [32][STRIDE]: row = event, F features + weight
  pipe.init();
  pipe.prologue();
  double acc[NP][2];
#pragma unroll
  for (int q = 0; q < NP; ++q) acc[q][0] = acc[q][1] = 0.0;
  const int w_slot = M.n_su + M.n_inst + M.n_terms;
  int64_t k = 0;
  for (int64_t tile = blockIdx.x; tile < pipe.n_tiles; tile += gridDim.x, ++k) {
    const double *st = reinterpret_cast<const double *>(pipe.wait(k));
    int64_t i = tile * TILE + tid;
    double2 col[KCMAX];
    double wj = 0.0;
    if (i < n) {
      staged_columns<KCMAX, TILE>(M, LP, st, tid, sT, lane, col);
      wj = weighted ? st[w_slot * TILE + tid] : 1.0;
    } else {
#pragma unroll
      for (int c = 0; c < KCMAX; ++c) col[c] = make_double2(0.0, 0.0);
    }
    __syncwarp();                                        // the warp's lineshape scratch is no longer read
    double *row = Xs + lane * STRIDE;
#pragma unroll
    for (int c = 0; c < KCMAX; ++c) *reinterpret_cast<double2 *>(row + 2 * c) = col[c];
    row[F] = wj;
    __syncwarp();
    const double *base = Xs + (lane & 3) * STRIDE + (lane >> 2);
#pragma unroll
    for (int grp = 0; grp < 8; ++grp) {                  // 4 events per MMA, 8 groups per warp tile
      const double *r = base + grp * 4 * STRIDE;
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
    __syncthreads();                                     // stage and scratch are free
    pipe.refill(k);
  }
  // block reduction in warp order (over the idle stages), block partial = upper 8x8 blocks of X^T W X
  double *Ws = reinterpret_cast<double *>(smem + 128);   // [WARPS][NB*NB][64]
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
  for (int e = tid; e < NB * NB * 64; e += TILE) {
    int bi = e / (NB * 64), bj = (e / 64) % NB;
    if (bi > bj) continue;
    double sum = 0.0;
#pragma unroll
    for (int wp = 0; wp < WARPS; ++wp) sum += Ws[wp * NB * NB * 64 + e];
    partials[(int64_t)blockIdx.x * NB * NB * 64 + e] = sum;
  }
  __threadfence();
  __syncthreads();
  if (tid == 0) last = atomicAdd(ticket, 1u) == gridDim.x - 1;
  __syncthreads();
  if (!last) return;
  __threadfence();
  // final pass: upper blocks summed over blocks in index order, staged in shared memory, then G
  double *XtX = Ws;                                      // [NB][NB][64], reused
  for (int e = tid; e < NB * NB * 64; e += TILE) {
    int bi = e / (NB * 64), bj = (e / 64) % NB;
    if (bi > bj) continue;
    double sum = 0.0;
    for (unsigned b = 0; b < gridDim.x; ++b) sum += __ldcg(partials + (int64_t)b * NB * NB * 64 + e);
    XtX[e] = sum;
  }
  __syncthreads();
  auto xtx = [&](int m, int nn) {                        // symmetric: only the upper triangle is ever read
    if (m > nn) { int tmp = m; m = nn; nn = tmp; }
    return XtX[((m >> 3) * NB + (nn >> 3)) * 64 + (m & 7) * 8 + (nn & 7)];
  };
  for (int q = tid; q < KC * KC; q += TILE) {
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
