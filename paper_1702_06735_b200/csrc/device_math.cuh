// device_math.cuh -- fp64 four-vector algebra, closed-form spin factors, barrier factors, lineshapes,
// Philox4x32-10 and Raubold-Lynch generation as __device__ functions (sm_100a).
// Formulas: SURVEY.md 8(c) O-3 .. O-9 (the paper prints none of them).
#pragma once
#include "tables.h"

namespace tddp4k {

struct V4 { double e, x, y, z; };

__device__ __forceinline__ V4 operator+(V4 a, V4 b) { return {a.e + b.e, a.x + b.x, a.y + b.y, a.z + b.z}; }
__device__ __forceinline__ V4 operator-(V4 a, V4 b) { return {a.e - b.e, a.x - b.x, a.y - b.y, a.z - b.z}; }
__device__ __forceinline__ V4 operator*(V4 a, double f) { return {a.e * f, a.x * f, a.y * f, a.z * f}; }
// Minkowski product, metric (+,-,-,-)
__device__ __forceinline__ double dot(V4 a, V4 b) { return a.e * b.e - a.x * b.x - a.y * b.y - a.z * b.z; }
// L1(p, q) = q - p (p.q)/p^2   (O-3)
__device__ __forceinline__ V4 L1(V4 p, V4 q, double p2) { return q - p * (dot(p, q) / p2); }

// eps4(a,b,c,d) = det[a|b|c|d] of contravariant components, eps_{0123} = +1 (O-3).
// Laplace expansion along the (E,x) and (y,z) row pairs.
__device__ __forceinline__ double eps4(V4 a, V4 b, V4 c, V4 d) {
  double s0 = a.e * b.x - a.x * b.e, s1 = a.e * c.x - a.x * c.e, s2 = a.e * d.x - a.x * d.e;
  double s3 = b.e * c.x - b.x * c.e, s4 = b.e * d.x - b.x * d.e, s5 = c.e * d.x - c.x * d.e;
  double c5 = c.y * d.z - c.z * d.y, c4 = b.y * d.z - b.z * d.y, c3 = b.y * c.z - b.z * c.y;
  double c2 = a.y * d.z - a.z * d.y, c1 = a.y * c.z - a.z * c.y, c0 = a.y * b.z - a.z * b.y;
  return s0 * c5 - s1 * c4 + s2 * c3 + s3 * c2 - s4 * c1 + s5 * c0;
}

// breakup momentum squared, factored form, clamped at 0 (O-3); M = sqrt(s)
__device__ __forceinline__ double breakup2(double M, double s, double ma, double mb) {
  double rad = (M - ma - mb) * (M + ma + mb) * (M + ma - mb) * (M - ma + mb);
  return rad > 0.0 ? rad / (4.0 * s) : 0.0;
}

// un-normalised Blatt-Weisskopf factor F_L(z) (O-5)
__device__ __forceinline__ double barrier(int L, double z) {
  if (L == 0) return 1.0;
  if (L == 1) return rsqrt_pos(1.0 + z);
  return rsqrt_pos(9.0 + 3.0 * z + z * z);
}

// parameter-free shape of the running width: g = q^(2L+1) F_L(z)^2 / sqrt(s), so that
// m0 Gamma(s) = gam * g with gam = m0^2 Gamma0 / (q0^(2L+1) F_L(z0)^2)   (O-6)
__device__ __forceinline__ double width_shape(int L, double q2, double z, double M) {
  double q = sqrt_pos(q2);
  if (L == 0) return q * rcp_normal(M);
  if (L == 1) return q * q2 * rcp_normal((1.0 + z) * M);
  return q * q2 * q2 * rcp_normal((9.0 + 3.0 * z + z * z) * M);
}

// closed-form spin factors (O-4), role vectors r0..r3 already gathered.  IEEE divisions and square roots here, in L1, in
// breakup2 and for the invariant-mass roots: these quantities are differences of nearly equal terms for events next to a
// threshold, and the full-size parity (1e-10 on every P_i of 10 M events) has no room for a second ulp there.  The
// branch-free forms (jit_shared.cuh) are used where the result only multiplies: barrier factors, width shape, the
// boosts and two-body decays of the generator.
__device__ __forceinline__ double spin_factor(int sf, V4 r0, V4 r1, V4 r2, V4 r3) {
  if (sf == SF_NONRES) return 1.0;
  if (sf <= SF_VV_D) {
    V4 p1 = r0 + r1, q1 = r0 - r1, p2 = r2 + r3, q2 = r2 - r3;
    V4 pD = p1 + p2, qD = p1 - p2;
    V4 v1 = L1(p1, q1, dot(p1, p1)), v2 = L1(p2, q2, dot(p2, p2));
    if (sf == SF_VV_S) return dot(v1, v2);
    if (sf == SF_VV_P) return eps4(pD, qD, v1, v2);
    double sD = dot(pD, pD);
    V4 d = L1(pD, qD, sD);
    return dot(d, v1) * dot(d, v2) - dot(d, d) * (1.0 / 3.0) * (dot(v1, v2) - dot(pD, v1) * dot(pD, v2) / sD);
  }
  V4 pV = r0 + r1, qV = r0 - r1;
  V4 pX = pV + r2, qX = pV - r2;
  V4 pD = pX + r3, qD = pX - r3;
  double sX = dot(pX, pX), sD = dot(pD, pD);
  V4 v = L1(pV, qV, dot(pV, pV));
  V4 d = L1(pD, qD, sD);
  if (sf == SF_AP_S) return -(dot(d, v) - dot(pX, d) * dot(pX, v) / sX);
  V4 t = L1(pX, qX, sX);
  // axial -> V P in D-wave: d_mu L2^{mu nu}(pX, qX) v_nu
  if (sf == SF_AP_D) return dot(d, t) * dot(t, v) - dot(t, t) * (1.0 / 3.0) * (dot(d, v) - dot(pX, d) * dot(pX, v) / sX);
  return dot(d, t) * eps4(d, t, pX, v) + dot(d, d) * (1.0 / 3.0) * (dot(pD, t) / sD) * eps4(pD, t, pX, v);
}

// ---------------------------------------------------------------------------------------------------
// Per-thread scratch in shared memory: row r of thread tid is base[r * stride + tid] (conflict-free).
struct Scratch {
  double *p;    // 16 rows: four-momenta of the event
  double *s;    // MAX_SYS rows: invariant masses squared
  double *q2;   // MAX_INST rows: breakup momentum squared of each instance's own decay
  int stride;
  __device__ __forceinline__ double &P(int r, int tid) const { return p[r * stride + tid]; }
  __device__ __forceinline__ double &S(int r, int tid) const { return s[r * stride + tid]; }
  __device__ __forceinline__ double &Q(int r, int tid) const { return q2[r * stride + tid]; }
  __device__ __forceinline__ V4 vec(int particle, int tid) const {
    return {P(4 * particle, tid), P(4 * particle + 1, tid), P(4 * particle + 2, tid), P(4 * particle + 3, tid)};
  }
};

// step 1 for one event whose momenta sit in scratch: invariant masses, shape functions, static factors.
// sink.s(i, v), sink.g(row, v), sink.f(row, v) receive the results (rows of the cache: InstTab::grow, TermTab::frow).
template <class Sink>
__device__ __forceinline__ void kinematics(const ModelTab &M, const Scratch &sc, int tid, Sink &sink) {
  for (int i = 0; i < M.n_sys; ++i) {
    unsigned mask = M.sys_mask[i];
    V4 sum = {0.0, 0.0, 0.0, 0.0};
    for (int a = 0; a < 4; ++a)
      if (mask & (1u << a)) sum = sum + sc.vec(a, tid);
    double s = dot(sum, sum);
    sc.S(i, tid) = s;
    sink.s(i, s);
  }
  for (int i = 0; i < M.n_inst; ++i) {
    const InstTab &in = M.inst[i];
    double s = sc.S(in.sys, tid);
    double Mr = sqrt(s);
    double ma = in.sub >= 0 ? sqrt(sc.S(in.sub, tid)) : in.ma;
    double q2 = breakup2(Mr, s, ma, in.mb);
    sc.Q(i, tid) = q2;
    sink.g(in.grow, in.kind == LS_CONSTANT ? 1.0 : width_shape(in.L, q2, q2 * in.r2, Mr));   // shared rows: same value again
  }
  double sD = sc.S(M.sysD, tid);
  double mD = sqrt(sD);
  for (int k = 0; k < M.n_terms; ++k) {
    const TermTab &tm = M.term[k];
    double f = 1.0;
    if (tm.sf != SF_NONRES) {
      V4 r0 = sc.vec(tm.perm[0], tid), r1 = sc.vec(tm.perm[1], tid);
      V4 r2 = sc.vec(tm.perm[2], tid), r3 = sc.vec(tm.perm[3], tid);
      f = spin_factor(tm.sf, r0, r1, r2, r3);
      const InstTab &i0 = M.inst[tm.inst0], &i1 = M.inst[tm.inst1];
      // D vertex: VV: D -> R1 R2 (both running); cascade: D -> X perm[3]
      double m1 = sqrt(sc.S(i0.sys, tid));
      double m2 = tm.sf <= SF_VV_D ? sqrt(sc.S(i1.sys, tid)) : M.m_final[tm.perm[3]];
      double qD2 = breakup2(mD, sD, m1, m2);
      f *= barrier(tm.LD, qD2 * M.r_parent2);
      f *= barrier(i0.L, sc.Q(tm.inst0, tid) * i0.r2);
      f *= barrier(i1.L, sc.Q(tm.inst1, tid) * i1.r2);
    }
    if (tm.frow >= 0) sink.f(tm.frow, f);    // a constant-amplitude term keeps no row (f = 1)
  }
}

// ---------------------------------------------------------------------------------------------------
// G1: Philox4x32-10 (O-9): counter (i_lo, i_hi, block, stream), key (seed_lo, seed_hi)
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                              uint32_t k1, uint32_t out[4]) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}
__device__ __forceinline__ void uniform_pair(uint64_t seed, uint64_t index, uint32_t block, uint32_t stream,
                                             double &u0, double &u1) {
  uint32_t w[4];
  philox4x32_10((uint32_t)index, (uint32_t)(index >> 32), block, stream, (uint32_t)seed, (uint32_t)(seed >> 32), w);
  uint64_t a = ((uint64_t)w[0] << 32) | w[1], b = ((uint64_t)w[2] << 32) | w[3];
  u0 = (double)(a >> 11) * 0x1.0p-53;
  u1 = (double)(b >> 11) * 0x1.0p-53;
}

__device__ __forceinline__ double breakup_excess(double excess, double M, double ma, double mb) {
  double rad = excess * (M + ma + mb) * (M + ma - mb) * (M - ma + mb);
  return rad > 0.0 ? div_normal(sqrt_pos(rad), 2.0 * M) : 0.0;
}
// E' = (E_P E + P.p)/M ; p' = p + P [ (P.p)/(M (E_P + M)) + E/M ]   (O-9)
__device__ __forceinline__ V4 boost(V4 P, double M, V4 p) {
  double Pp = P.x * p.x + P.y * p.y + P.z * p.z;
  const double iM = rcp_normal(M);
  double f = div_normal(Pp, M * (P.e + M)) + div_by(p.e, iM, M);
  return {div_by(P.e * p.e + Pp, iM, M), p.x + P.x * f, p.y + P.y * f, p.z + P.z * f};
}
__device__ __forceinline__ void two_body(double m_first, double m_second, double ps, double u_cos, double u_phi,
                                         V4 &first, V4 &second) {
  double ct = 2.0 * u_cos - 1.0;
  double st = sqrt_pos(1.0 - ct * ct);
  double sphi, cphi;
  sincospi(2.0 * u_phi, &sphi, &cphi);   // phi = 2 pi u: exact argument reduction, no multiple-of-pi rounding
  double nx = st * cphi, ny = st * sphi, nz = ct;
  first = {sqrt_pos(m_first * m_first + ps * ps), ps * nx, ps * ny, ps * nz};
  second = {sqrt_pos(m_second * m_second + ps * ps), -ps * nx, -ps * ny, -ps * nz};
}
// G2/G3: one Raubold-Lynch candidate (O-9).  p[0..3]: final-state momenta in the D rest frame.
__device__ __forceinline__ void rl_candidate(const double (&mf)[4], double m_parent, double tau, uint64_t seed, uint32_t stream,
                                             uint64_t i, V4 p[4], double &t, double &w, double &u_acc) {
  double ra, rb, c1, f1, c2, f2, c3, f3, ut;
  uniform_pair(seed, i, 0, stream, ra, rb);
  uniform_pair(seed, i, 1, stream, c1, f1);
  uniform_pair(seed, i, 2, stream, c2, f2);
  uniform_pair(seed, i, 3, stream, c3, f3);
  uniform_pair(seed, i, 4, stream, ut, u_acc);
  double r1 = fmin(ra, rb), r2 = fmax(ra, rb);
  double Tk = m_parent - (mf[0] + mf[1] + mf[2] + mf[3]);
  double M2 = mf[0] + mf[1] + r1 * Tk, M3 = mf[0] + mf[1] + mf[2] + r2 * Tk, M4 = m_parent;
  double ps1 = breakup_excess((1.0 - r2) * Tk, M4, M3, mf[3]);
  double ps2 = breakup_excess((r2 - r1) * Tk, M3, M2, mf[2]);
  double ps3 = breakup_excess(r1 * Tk, M2, mf[0], mf[1]);
  V4 X3, X2, a, b, tmp;
  two_body(M3, mf[3], ps1, c1, f1, X3, p[3]);
  two_body(M2, mf[2], ps2, c2, f2, X2, tmp);
  p[2] = boost(X3, M3, tmp);
  two_body(mf[0], mf[1], ps3, c3, f3, a, b);
  p[0] = boost(X3, M3, boost(X2, M2, a));
  p[1] = boost(X3, M3, boost(X2, M2, b));
  w = ps1 * ps2 * ps3;
  t = -tau * log(1.0 - ut);
}

}  // namespace tddp4k
