// kernels.cuh -- the CUDA kernels of the hot path, sm_100a, fp64.
// All kernels take their tables by value (__grid_constant__): no global state, any stream, any handle.
#pragma once
#include <stdint.h>
#include "device_math.cuh"

namespace tddp4k {

// ------------------------------------------------------------------------------------------------
// deterministic block reductions (fixed shuffle tree, then warp 0 over the warp partials)
template <int BLOCK>
__device__ __forceinline__ double block_sum(double v, double *red /* [BLOCK/32] shared */) {
  v = warp_sum(v);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
  __syncthreads();
  double r = 0.0;
  if (threadIdx.x < 32) {
    r = threadIdx.x < BLOCK / 32 ? red[threadIdx.x] : 0.0;
    r = warp_sum(r);
  }
  return r;  // valid in warp 0
}

// ------------------------------------------------------------------------------------------------
// step 1: kinematics + spin factors, once per event set.  One thread per event.
// in : p4 rows [16][ld_in];  out: the tile-major static cache (tables.h): rows s [n_sys], g from g_row0, f from f_row0
constexpr int KIN_BLOCK = 128;
struct CacheRows { int R, g_row0, f_row0; };
__device__ __forceinline__ int64_t tile_index(int R, int row, int64_t i) { return ((i >> 5) * R + row) * 32 + (i & 31); }
struct KinSink {
  double *cache;
  CacheRows cr;
  int64_t i;
  __device__ __forceinline__ void s(int r, double v) { cache[tile_index(cr.R, r, i)] = v; }
  __device__ __forceinline__ void g(int r, double v) { cache[tile_index(cr.R, cr.g_row0 + r, i)] = v; }
  __device__ __forceinline__ void f(int r, double v) { cache[tile_index(cr.R, cr.f_row0 + r, i)] = v; }
};
__global__ void __launch_bounds__(KIN_BLOCK)
kin_kernel(const __grid_constant__ ModelTab M, const double *__restrict__ p4, int64_t ld_in, int64_t n,
           double *__restrict__ cache, CacheRows cr) {
  extern __shared__ double smem[];
  Scratch sc{smem, smem + 16 * KIN_BLOCK, smem + (16 + M.n_sys) * KIN_BLOCK, KIN_BLOCK};
  int tid = threadIdx.x;
  int64_t i = (int64_t)blockIdx.x * KIN_BLOCK + tid;
  if (i >= n) return;
#pragma unroll
  for (int r = 0; r < 16; ++r) sc.P(r, tid) = p4[r * ld_in + i];
  KinSink sink{cache, cr, i};
  kinematics(M, sc, tid, sink);
}
__global__ void __launch_bounds__(256) fill_kernel(double *__restrict__ dst, int64_t n, double v) {
  int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
  if (i < n) dst[i] = v;
}
// one row of the tile-major cache <-> a plain vector (weights in at load; inspection rows out)
__global__ void __launch_bounds__(256) row_scatter_kernel(double *__restrict__ cache, int R, int row, int64_t n,
                                                         const double *__restrict__ src) {
  int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
  if (i < n) cache[tile_index(R, row, i)] = src[i];
}
__global__ void __launch_bounds__(256) row_gather_kernel(const double *__restrict__ cache, int R, int row, int64_t n,
                                                        double *__restrict__ dst) {
  int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
  if (i < n) dst[i] = cache[tile_index(R, row, i)];
}

// ------------------------------------------------------------------------------------------------
// Validation observables of the paper's Fig. 3: m12, m34, cos12, cos34, phi with 12 = (pi+ pi-) =
// particles (2,3) and 34 = (K+ pi-) = (0,1).  Frame-independent forms, no boosts: with P the pair, a its
// first daughter, S the other pair,  cos = -[(a.P)(S.P)/P^2 - a.S] / sqrt{[(a.P)^2/P^2 - a^2] [(S.P)^2/P^2 - S^2]};
// with a = p2, b = p0 projected orthogonally to the plane spanned by D = P12 + P34 and P12 (Gram form),
// cos phi = a_perp.b_perp / sqrt(a_perp^2 b_perp^2),  sin phi = -eps4(D, P12, a, b) / sqrt{[(D.P12)^2 - D^2 P12^2] a_perp^2 b_perp^2}.
// One thread per event; integer histogram counts (exact, order-independent) through shared-memory atomics.
constexpr int PROJ_BLOCK = 256, PROJ_MAX_BINS = 512;
struct ProjRanges { double lo[5], inv_width[5], hi[5]; };
__device__ __forceinline__ double helicity_cos(V4 a, V4 P, V4 S, double sP, double sS) {
  double aP = dot(a, P), SP = dot(S, P);
  double num = aP * SP / sP - dot(a, S);
  double ka2 = aP * aP / sP - dot(a, a), ks2 = SP * SP / sP - sS;
  return -num / sqrt(ka2 * ks2);
}
__global__ void __launch_bounds__(PROJ_BLOCK)
project_kernel(const double *__restrict__ p4, int64_t ld, int64_t n, int n_bins, const __grid_constant__ ProjRanges R,
               unsigned long long *__restrict__ hist /* [5][n_bins] */, double *__restrict__ values /* [5][n] or NULL */) {
  __shared__ unsigned int s_h[5 * PROJ_MAX_BINS];
  for (int k = threadIdx.x; k < 5 * n_bins; k += PROJ_BLOCK) s_h[k] = 0u;
  __syncthreads();
  const int64_t stride = (int64_t)gridDim.x * PROJ_BLOCK;
  for (int64_t i = (int64_t)blockIdx.x * PROJ_BLOCK + threadIdx.x; i < n; i += stride) {
    V4 p[4];
#pragma unroll
    for (int a = 0; a < 4; ++a) p[a] = {p4[(4 * a) * ld + i], p4[(4 * a + 1) * ld + i], p4[(4 * a + 2) * ld + i], p4[(4 * a + 3) * ld + i]};
    const V4 P12 = p[2] + p[3], P34 = p[0] + p[1], D = P12 + P34;
    const double s12 = dot(P12, P12), s34 = dot(P34, P34), sD = dot(D, D), DP = dot(D, P12);
    double v[5];
    v[0] = sqrt(s12);
    v[1] = sqrt(s34);
    v[2] = helicity_cos(p[2], P12, P34, s12, s34);
    v[3] = helicity_cos(p[0], P34, P12, s34, s12);
    const double den = sD * s12 - DP * DP;                       // < 0: -(M_D |P12 vec|)^2 in the D rest frame
    auto perp = [&](V4 a, V4 b) {
      double aD = dot(a, D), bD = dot(b, D), aP = dot(a, P12), bP = dot(b, P12);
      return dot(a, b) - (aD * bD * s12 - aD * bP * DP - aP * bD * DP + aP * bP * sD) / den;
    };
    const double aa = perp(p[2], p[2]), bb = perp(p[0], p[0]), ab = perp(p[2], p[0]);
    const double nrm = sqrt(aa * bb);
    v[4] = atan2(-eps4(D, P12, p[2], p[0]) / (sqrt(-den) * nrm), ab / nrm);
#pragma unroll
    for (int k = 0; k < 5; ++k) {
      if (values) values[(int64_t)k * n + i] = v[k];
      int b = (int)floor((v[k] - R.lo[k]) * R.inv_width[k] * n_bins);
      if (v[k] == R.hi[k]) b = n_bins - 1;
      if (b >= 0 && b < n_bins) atomicAdd(&s_h[k * n_bins + b], 1u);
    }
  }
  __syncthreads();
  for (int k = threadIdx.x; k < 5 * n_bins; k += PROJ_BLOCK)
    if (s_h[k]) atomicAdd(&hist[k], (unsigned long long)s_h[k]);
}

// ------------------------------------------------------------------------------------------------
// Sum of the ranks' Gram sums in rank order (event-sharded evaluation): gathered [world][len]
__global__ void __launch_bounds__(256) gram_reduce_kernel(const double *__restrict__ gathered, int world, int stride, int len,
                                                         double *__restrict__ G) {
  for (int q = threadIdx.x; q < len; q += 256) {
    double sum = 0.0;
    for (int r = 0; r < world; ++r) sum += gathered[(int64_t)r * stride + q];
    G[q] = sum;
  }
}
__global__ void __launch_bounds__(32) append_count_kernel(double *dst, double value) { if (threadIdx.x == 0) *dst = value; }

// fp64 issue-rate probe: 8 independent DFMA chains per thread, 4096 FMAs each, 148 x 4 x 256 threads
// The branch-free fp64 primitives of jit_shared.cuh on arrays (tddp4_math_probe): what = 0 rcp_normal(x), 1 sqrt_pos(x),
// 2 rsqrt_pos(x), 3 div_normal(x, y).  For the accuracy tests only.
__global__ void __launch_bounds__(256) math_probe_kernel(int what, int64_t n, const double *__restrict__ x,
                                                         const double *__restrict__ y, double *__restrict__ out) {
  int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
  if (i >= n) return;
  double v = x[i];
  out[i] = what == 0 ? rcp_normal(v) : what == 1 ? sqrt_pos(v) : what == 2 ? rsqrt_pos(v) : div_normal(v, y[i]);
}

__global__ void __launch_bounds__(256) fp64_peak_kernel(double *out, double a, double b, int iters) {
  double v[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) v[k] = a + k + threadIdx.x;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 16; ++r)
#pragma unroll
      for (int k = 0; k < 8; ++k) v[k] = fma(v[k], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int k = 0; k < 8; ++k) s += v[k];
  if (s == 123.456) out[0] = s;
}

// ------------------------------------------------------------------------------------------------
constexpr int COL_BLOCK = 128;
// per-term amplitudes a_k (un-summed), for per-layer parity only (TDDP4_GET_TERMS)
__global__ void __launch_bounds__(COL_BLOCK)
terms_kernel(const __grid_constant__ ModelTab M, const __grid_constant__ LineParams LP, const double *__restrict__ cache,
             CacheRows cr, int64_t n, double2 *__restrict__ out /* [n_terms][n], caller's term order */) {
  extern __shared__ double2 sT[];
  int tid = threadIdx.x;
  int64_t i = (int64_t)blockIdx.x * COL_BLOCK + tid;
  if (i >= n) return;
  for (int j = 0; j < M.n_inst; ++j)
    sT[j * COL_BLOCK + tid] = breit_wigner(LP.m0sq[j], LP.gam[j], cache[tile_index(cr.R, M.inst[j].sys, i)],
                                           cache[tile_index(cr.R, cr.g_row0 + M.inst[j].grow, i)]);
  for (int k = 0; k < M.n_terms; ++k) {
    const TermTab &tm = M.term[k];
    double fv = tm.frow >= 0 ? cache[tile_index(cr.R, cr.f_row0 + tm.frow, i)] : 1.0;
    double2 T = make_double2(1.0, 0.0);
    if (tm.inst0 >= 0) T = cmul(sT[tm.inst0 * COL_BLOCK + tid], sT[tm.inst1 * COL_BLOCK + tid]);
    out[(int64_t)M.user_term[k] * n + i] = make_double2(fv * T.x, fv * T.y);
  }
}

// ------------------------------------------------------------------------------------------------
// deterministic sum, max |.| and minimum of a vector (decay times, sigma_t at load): one block, fixed order
__global__ void __launch_bounds__(1024) stat_kernel(const double *__restrict__ v, int64_t n, double *out /* [3] */) {
  __shared__ double red[32];
  __shared__ double red2[32];
  double acc = 0.0, mx = 0.0, mn = INFINITY;
  for (int64_t i = threadIdx.x; i < n; i += 1024) {
    double x = v[i];
    acc += x;
    mx = fmax(mx, fabs(x));
    mn = fmin(mn, x);
  }
  acc = block_sum<1024>(acc, red);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    mn = fmin(mn, __shfl_xor_sync(0xffffffffu, mn, o));
  }
  __syncthreads();
  if ((threadIdx.x & 31) == 0) { red[threadIdx.x >> 5] = mx; red2[threadIdx.x >> 5] = mn; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int k = 1; k < 32; ++k) { mx = fmax(mx, red[k]); mn = fmin(mn, red2[k]); }
    out[0] = acc;
    out[1] = mx;
    out[2] = mn;
  }
}

}  // namespace tddp4k
#include "stream_kernels.cuh"
namespace tddp4k {

// ------------------------------------------------------------------------------------------------
// G1-G5: candidate generation with the rate evaluated on the fly is the run-time specialised kernel of gen_jit.cuh
// (one thread per candidate, GEN_BLOCK candidates per block: flags and block counts below are laid out for it).
constexpr int GEN_BLOCK = 128;

// Output offsets of one launch chunk, one per span of EMIT_SPAN candidates (= SCAN_PER ratio blocks; an emit block covers
// one span), continued from the running total of the chunks before it: offs[s] = *total + number of accepted candidates in
// the spans before s; *total advances by the chunk's count (no host round trip).  Single block: a thread sums the
// SCAN_PER counts of its span (four 16-byte loads), the block scans the span sums with warp shuffles in tiles of 1024 spans
// and carries the running total from tile to tile; the next tile's counts are loaded before the current tile is scanned.
// Integer arithmetic: the same result in any order.  (The first version scanned every block count, each thread one
// contiguous stretch and thread 0 the 1024 stretch sums serially: 63 us for the 78 125 counts of config 4, 234 us for a
// 16 M-candidate chunk -- a tenth of the generation time.)
constexpr int EMIT_BLOCK = 128, EMIT_SPAN = 2048, EMIT_WORDS = EMIT_SPAN / 32;
static_assert(EMIT_SPAN % GEN_BLOCK == 0, "an emit block starts at a ratio-block boundary");
constexpr int SCAN_BLOCK = 1024, SCAN_PER = EMIT_SPAN / GEN_BLOCK;
static_assert(SCAN_PER % 4 == 0, "a span's counts are loaded as uint4");
__global__ void __launch_bounds__(SCAN_BLOCK) scan_kernel(const uint32_t *__restrict__ cnt /* allocated in whole spans */, int64_t n_blocks,
                                                          unsigned long long *__restrict__ offs /* [n_spans] */,
                                                          unsigned long long *__restrict__ total) {
  __shared__ uint32_t s_warp[SCAN_BLOCK / 32];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  unsigned long long carry = *total;
  const int64_t n_spans = (n_blocks + SCAN_PER - 1) / SCAN_PER;
  auto span_sum = [&](int64_t sp) -> uint32_t {
    if (sp >= n_spans) return 0u;
    const int64_t b = sp * SCAN_PER;
    const uint4 *src = reinterpret_cast<const uint4 *>(cnt + b);
    uint32_t acc = 0;
#pragma unroll
    for (int k = 0; k < SCAN_PER / 4; ++k) {               // counts beyond this chunk's blocks are leftovers of a larger chunk
      uint4 q = src[k];
      const int64_t r = n_blocks - (b + 4 * k);            // blocks left from this quad on
      acc += (r > 0 ? q.x : 0u) + (r > 1 ? q.y : 0u) + (r > 2 ? q.z : 0u) + (r > 3 ? q.w : 0u);
    }
    return acc;
  };
  uint32_t next = span_sum(tid);
  for (int64_t s0 = 0; s0 < n_spans; s0 += SCAN_BLOCK) {
    const uint32_t mine = next;
    next = span_sum(s0 + SCAN_BLOCK + tid);                 // in flight while this tile is scanned
    uint32_t incl = mine;                                   // inclusive scan over the warp
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      uint32_t y = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += y;
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    if (warp == 0) {                                        // inclusive scan of the 32 warp totals
      uint32_t w = s_warp[lane];
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        uint32_t y = __shfl_up_sync(0xffffffffu, w, o);
        if (lane >= o) w += y;
      }
      s_warp[lane] = w;
    }
    __syncthreads();
    if (s0 + tid < n_spans) offs[s0 + tid] = carry + (warp ? s_warp[warp - 1] : 0u) + (incl - mine);
    carry += s_warp[SCAN_BLOCK / 32 - 1];
    __syncthreads();                                        // s_warp is reused by the next tile
  }
  if (tid == 0) *total = carry;
}

// G6: regenerate the accepted candidates (Philox is counter based: no state to carry) and write them compacted, in
// candidate order.  One block covers EMIT_SPAN candidates: it first turns their accept bits into a dense list of local
// indices in shared memory, then its threads walk that list, so every lane that runs Philox + Raubold-Lynch produces an
// output event (at 6.6 % acceptance the one-thread-per-candidate form kept 89 % of the warps busy for 1/15 of the
// lanes: 0.96 ms against 1.21 ms for the ratio pass itself) and consecutive threads write consecutive output slots.
__global__ void __launch_bounds__(EMIT_BLOCK)
gen_emit_kernel(const __grid_constant__ ModelTab M, double tau, uint64_t seed, uint32_t stream, uint64_t first,
                int64_t n, const uint32_t *__restrict__ flags, const unsigned long long *__restrict__ offs,
                int64_t capacity, double *__restrict__ out_p4, double *__restrict__ out_t,
                int64_t *__restrict__ out_index) {
  __shared__ uint16_t s_list[EMIT_SPAN];
  __shared__ int s_pre[EMIT_WORDS + 1];
  const int tid = threadIdx.x;
  const int64_t j0 = (int64_t)blockIdx.x * EMIT_SPAN;
  uint32_t word = 0;
  if (tid < EMIT_WORDS && j0 + (int64_t)tid * 32 < n) word = flags[(j0 >> 5) + tid];
  if (tid < EMIT_WORDS) s_pre[tid + 1] = __popc(word);
  if (tid == 0) s_pre[0] = 0;
  __syncthreads();
  if (tid == 0)
    for (int k = 1; k <= EMIT_WORDS; ++k) s_pre[k] += s_pre[k - 1];
  __syncthreads();
  if (tid < EMIT_WORDS) {
    int at = s_pre[tid];
    while (word) {
      int b = __ffs(word) - 1;
      word &= word - 1;
      s_list[at++] = (uint16_t)(tid * 32 + b);
    }
  }
  __syncthreads();
  const int count = s_pre[EMIT_WORDS];
  const int64_t base = (int64_t)offs[blockIdx.x];
  for (int k = tid; k < count; k += EMIT_BLOCK) {
    const int64_t pos = base + k;
    if (pos >= capacity) break;
    const int64_t j = j0 + s_list[k];
    V4 p[4];
    double t, w, u;
    rl_candidate(M.m_final, M.m_parent, tau, seed, stream, first + (uint64_t)j, p, t, w, u);
    if (out_p4) {
#pragma unroll
      for (int a = 0; a < 4; ++a) {
        out_p4[(4 * a) * capacity + pos] = p[a].e; out_p4[(4 * a + 1) * capacity + pos] = p[a].x;
        out_p4[(4 * a + 2) * capacity + pos] = p[a].y; out_p4[(4 * a + 3) * capacity + pos] = p[a].z;
      }
    }
    if (out_t) out_t[pos] = t;
    if (out_index) out_index[pos] = (int64_t)first + j;
  }
}

}  // namespace tddp4k
