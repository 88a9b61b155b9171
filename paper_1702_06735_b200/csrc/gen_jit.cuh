// gen_jit.cuh -- G1-G5 of the generation path (phase-space events "weighted by the
// decay rate", accept / reject): one thread per Raubold-Lynch candidate draws its Philox numbers, builds the four momenta
// and the decay time (O-9), evaluates the kinematics, spin factors, lineshapes and amplitudes of the model on the fly
// (nothing is cached for a candidate that is seen once) and the rate of eq. (1), and either dumps the candidate (mode 0,
// parity), feeds the exact pilot maximum (mode 1, G5) or writes one accept bit and the per-block counts (mode 2, G6).
//
// NOT compiled by nvcc: compiled at run time with NVRTC (jit.h) behind the generated prelude, which states the model --
// particle systems, lineshape instances, terms, masses, radii -- as compile-time constants (J_*).  The table-driven form
// of round 1 kept momenta, invariant masses, breakup momenta and lineshapes of a candidate in per-thread shared-memory
// rows (the tables index them at run time): 128 registers, 6 warps per SM, every sqrt(s) recomputed at each use.  Here
// every index is an immediate, everything lives in registers, and common subexpressions (the root of each invariant
// mass, each breakup momentum) are computed once.
#include "device_math.cuh"

namespace tddp4k {

constexpr int GEN_BLOCK = 128;

// steps 1-5 for one candidate in registers; formulas as kinematics() of device_math.cuh (O-3 .. O-6)
__device__ __forceinline__ double candidate_ratio(const LineParams &LP, const RateParams &R, const V4 (&p)[4], double t, double w) {
  double s[J_NSYS], rs[J_NSYS];
#pragma unroll
  for (int i = 0; i < J_NSYS; ++i) {
    V4 sum = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
    for (int a = 0; a < 4; ++a)
      if (J_SYSMASK[i] & (1 << a)) sum = sum + p[a];
    s[i] = dot(sum, sum);
    rs[i] = sqrt(s[i]);   // IEEE: M - m_a - m_b cancels near a threshold, where half an ulp of M matters
  }
  double q2[J_NINST + 1];
  double2 T[J_NINST + 1];
#pragma unroll
  for (int j = 0; j < J_NINST; ++j) {
    const double sj = s[J_INST_SYS[j]], Mr = rs[J_INST_SYS[j]];
    const double ma = J_INST_SUB[j] >= 0 ? rs[J_INST_SUB[j] >= 0 ? J_INST_SUB[j] : 0] : J_INST_MA[j];
    q2[j] = breakup2(Mr, sj, ma, J_INST_MB[j]);
    const double g = J_INST_KIND[j] == LS_CONSTANT ? 1.0 : width_shape(J_INST_L[j], q2[j], q2[j] * J_INST_R2[j], Mr);
    T[j] = breit_wigner(LP.m0sq[j], LP.gam[j], sj, g);
  }
  const double sD = s[J_SYSD], mD = rs[J_SYSD];
  double2 A = make_double2(0.0, 0.0), Ab = make_double2(0.0, 0.0), col = make_double2(0.0, 0.0);
#pragma unroll
  for (int k = 0; k < J_NTERMS; ++k) {
    double f = 1.0;
    double2 P = make_double2(1.0, 0.0);
    if (J_TERM_SF[k] != SF_NONRES) {
      const int i0 = J_T0[k] >= 0 ? J_T0[k] : 0, i1 = J_T1[k] >= 0 ? J_T1[k] : 0;
      f = spin_factor(J_TERM_SF[k], p[J_TERM_P0[k]], p[J_TERM_P1[k]], p[J_TERM_P2[k]], p[J_TERM_P3[k]]);
      // D vertex: VV: D -> R1 R2 (both running); cascade: D -> X perm[3]
      const double m1 = rs[J_INST_SYS[i0]];
      const double m2 = J_TERM_SF[k] <= SF_VV_D ? rs[J_INST_SYS[i1]] : J_MFINAL[J_TERM_P3[k]];
      const double qD2 = breakup2(mD, sD, m1, m2);
      f *= barrier(J_TERM_LD[k], qD2 * J_RPARENT2);
      f *= barrier(J_INST_L[i0], q2[i0] * J_INST_R2[i0]);
      f *= barrier(J_INST_L[i1], q2[i1] * J_INST_R2[i1]);
      P = cmul(T[i0], T[i1]);
    }
    col.x = fma(f, P.x, col.x);
    col.y = fma(f, P.y, col.y);
    if (J_LAST[k]) {
      amp_add(A, Ab, R.c[J_COL[k]][0], R.c[J_COL[k]][1], R.cbar[J_COL[k]][0], R.cbar[J_COL[k]][1], col);
      col = make_double2(0.0, 0.0);
    }
  }
  return w * bracket<false>(A, Ab, R.y * R.Gamma * t, R.x * R.Gamma * t);
}

// mode 0: raw candidate dump (parity); mode 1: pilot maximum (G5); mode 2: accept flags + block counts (G6)
extern "C" __global__ void __launch_bounds__(GEN_BLOCK, J_GEN_BPS)
gen_jit(const __grid_constant__ LineParams LP, const __grid_constant__ RateParams R, double tau, unsigned long long seed,
        unsigned int stream, unsigned long long first, long long n, int mode,
        double envelope /* mode 2: the envelope, or its scale if from_pilot */, int from_pilot,
        double *__restrict__ out_p4, double *__restrict__ out_t, double *__restrict__ out_w,
        double *__restrict__ out_ratio, double *__restrict__ out_u,
        unsigned long long *pilot_max_bits, unsigned int *__restrict__ flags /* one bit per candidate */,
        unsigned int *__restrict__ block_count, unsigned long long *overflow) {
  __shared__ int s_cnt[GEN_BLOCK / 32];
  const int tid = threadIdx.x;
  const long long j = (long long)blockIdx.x * GEN_BLOCK + tid;
  const bool live = j < n;
  V4 p[4];
  double t = 0.0, w = 0.0, u = 1.0, rho = 0.0;
  if (live) {
    const double mf[4] = {J_MFINAL[0], J_MFINAL[1], J_MFINAL[2], J_MFINAL[3]};
    rl_candidate(mf, J_MPARENT, tau, seed, stream, first + (unsigned long long)j, p, t, w, u);
    rho = candidate_ratio(LP, R, p, t, w);
  }
  if (mode == 0) {
    if (!live) return;
    if (out_p4) {
#pragma unroll
      for (int a = 0; a < 4; ++a) {
        out_p4[(4 * a) * n + j] = p[a].e; out_p4[(4 * a + 1) * n + j] = p[a].x;
        out_p4[(4 * a + 2) * n + j] = p[a].y; out_p4[(4 * a + 3) * n + j] = p[a].z;
      }
    }
    if (out_t) out_t[j] = t;
    if (out_w) out_w[j] = w;
    if (out_ratio) out_ratio[j] = rho;
    if (out_u) out_u[j] = u;
    return;
  }
  if (mode == 1) {
    // rho >= 0: the IEEE bit pattern is monotone, so an integer max is the exact fp64 max
    double m = live && rho > 0.0 ? rho : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((tid & 31) == 0) atomicMax(pilot_max_bits, (unsigned long long)__double_as_longlong(m));
    return;
  }
  if (from_pilot) envelope *= __longlong_as_double((long long)*pilot_max_bits);   // E = scale * max over the pilot (G5), no host round trip
  const bool acc = live && (u * envelope < rho);
  const unsigned ballot = __ballot_sync(0xffffffffu, acc);
  const unsigned over = __ballot_sync(0xffffffffu, live && rho > envelope);
  if ((tid & 31) == 0) {
    flags[j >> 5] = ballot;
    s_cnt[tid >> 5] = __popc(ballot);
    if (over) atomicAdd(overflow, (unsigned long long)__popc(over));
  }
  __syncthreads();
  if (tid == 0) {
    int c = 0;
#pragma unroll
    for (int k = 0; k < GEN_BLOCK / 32; ++k) c += s_cnt[k];
    block_count[blockIdx.x] = c;
  }
}

}  // namespace tddp4k
