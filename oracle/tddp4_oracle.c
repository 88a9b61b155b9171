/*
 * tddp4_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU restatement of the time-dependent D0 -> K+ pi- pi+ pi-
 * likelihood of arXiv:1702.06735 and of its companion event generator.  It is
 * written from the paper (cited as P:<line> of /root/reference/PAPER.md) and, where
 * the paper prints no formula, from the readings fixed in SURVEY.md 8(c)
 * (cited as O-1 .. O-9) and listed in DESIGN.md.  Only tests/, bench.py's
 * cpu_baseline / --impl reference legs and __graft_entry__.smoke() may call it.
 *
 * It shares no code, header, table or constant with the CUDA path
 * (paper_1702_06735_b200/csrc).  Nothing here is cached, blocked, fused or
 * re-ordered: every call recomputes every quantity from the four-momenta, spin
 * factors are evaluated as explicit Lorentz-index loops, sums are Neumaier
 * compensated sums taken in event order.  OpenMP is used over events only (each
 * event writes its own output slot; reductions are done serially afterwards, so
 * results do not depend on the thread count).
 *
 * Parity pins (tests/test_oracle_*.py): Philox stream vs cuRAND's host Philox4_32_10;
 * momentum conservation, mass shells, massless 4-body volume pi^3 M^4/96; T(m0^2) =
 * i/(m0 Gamma0); Lorentz invariance, rest-frame reductions and closed forms of the spin
 * factors; special cases of eq. (1); time integrals vs quadrature; 10-event brute force
 * in mpmath.  "parity unpinned": that the conventions of O-3..O-7 are the ones
 * GooFit/MINT use (no reference values exist in the container).
 *
 * Units: GeV, ps.  Metric (+,-,-,-).  Four-vectors are (E, px, py, pz).
 * Final-state order: 0 = K+, 1 = pi-, 2 = pi+, 3 = pi- (O-3).
 * SoA event layout: p4[(4*particle + component) * n + event].
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_MAX_RES 16
#define ORC_MAX_TERMS 64
#define ORC_MAX_COUPLINGS 32

/* spin-factor kinds, O-4 */
enum { ORC_SF_NONRES = 0, ORC_SF_VV_S = 1, ORC_SF_VV_P = 2, ORC_SF_VV_D = 3, ORC_SF_AP_S = 4, ORC_SF_TP_D = 5,
       ORC_SF_AP_D = 6 };
/* lineshape kinds ("resonance lineshapes" is a class of building blocks; the paper names none) */
enum { ORC_LS_RUNNING = 0,   /* O-6: relativistic Breit-Wigner with mass-dependent width          */
       ORC_LS_CONSTANT = 1 };/* relativistic Breit-Wigner with constant width: 1/(m0^2 - s - i m0 Gamma0) */

typedef struct {
  double m_parent;            /* nominal D0 mass (used by the generator only)           */
  double m_final[4];          /* K+, pi-, pi+, pi-                                       */
  double r_res, r_parent;     /* Blatt-Weisskopf radii, GeV^-1 (O-5)                     */
  double t_lo, t_hi;          /* decay-time window; t_hi may be +inf (O-8)               */
  int n_res;
  int res_L[ORC_MAX_RES];     /* L of the resonance's own decay vertex (O-5)             */
  int n_terms;
  int term_sf[ORC_MAX_TERMS];        /* spin-factor kind                                 */
  int term_res[ORC_MAX_TERMS][2];    /* VV: {R1 on (r0,r1), R2 on (r2,r3)};
                                        cascade: {X on (r0,r1,r2), V on (r0,r1)}; -1 none */
  int term_perm[ORC_MAX_TERMS][4];   /* role r -> final-state index                      */
  int term_coupling[ORC_MAX_TERMS];  /* kappa(k): index of the coupling, O-2             */
  int n_couplings;
  double res_r[ORC_MAX_RES];  /* Blatt-Weisskopf radius of this resonance's own decay vertex; 0: r_res (O-5:    */
                              /* "per-resonance radii")                                     */
  int res_kind[ORC_MAX_RES];  /* ORC_LS_*                                                                       */
} orc_model;

typedef struct {
  double c[ORC_MAX_COUPLINGS][2];     /* couplings of A_f   (re, im), eq. (2)    */
  double cbar[ORC_MAX_COUPLINGS][2];  /* couplings of Abar_f                             */
  double mass[ORC_MAX_RES];           /* m0                                              */
  double width[ORC_MAX_RES];          /* Gamma0                                          */
  double x, y, tau;                   /* mixing parameters and lifetime, eq. (1) */
} orc_params;

/* ------------------------------------------------------------------------------------ */
/* Compensated summation (Neumaier), used for every sum over events.       */
typedef struct { double s, c; } orc_acc;
static void acc_add(orc_acc *a, double v) {
  double t = a->s + v;
  if (fabs(a->s) >= fabs(v)) a->c += (a->s - t) + v; else a->c += (v - t) + a->s;
  a->s = t;
}
static double acc_value(const orc_acc *a) { return a->s + a->c; }

double orc_sum(int64_t n, const double *v) {
  orc_acc a = {0.0, 0.0};
  for (int64_t i = 0; i < n; ++i) acc_add(&a, v[i]);
  return acc_value(&a);
}

int orc_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* ------------------------------------------------------------------------------------ */
/* O-9 / G1: Philox4x32-10 (Salmon et al., SC'11).  Ten rounds; the key is bumped by the  */
/* Weyl constants between rounds.                                                         */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    uint64_t p0 = (uint64_t)M0 * c0, p1 = (uint64_t)M1 * c2;
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += W0; k1 += W1;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* O-9: counter = (i_lo, i_hi, block, stream), key = (seed_lo, seed_hi); each block gives  */
/* two doubles u = ((w0*2^32 + w1) >> 11) * 2^-53 in [0,1).                                */
void orc_uniform_pair(uint64_t seed, uint64_t index, uint32_t block, uint32_t stream, double u[2]) {
  uint32_t ctr[4] = {(uint32_t)index, (uint32_t)(index >> 32), block, stream};
  uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  uint32_t w[4];
  orc_philox4x32_10(ctr, key, w);
  uint64_t a = ((uint64_t)w[0] << 32) | w[1], b = ((uint64_t)w[2] << 32) | w[3];
  u[0] = (double)(a >> 11) * 0x1.0p-53;
  u[1] = (double)(b >> 11) * 0x1.0p-53;
}

/* ------------------------------------------------------------------------------------ */
/* O-3: breakup momentum, factored form, radicand clamped at 0.                           */
double orc_breakup(double M, double ma, double mb) {
  double rad = (M - ma - mb) * (M + ma + mb) * (M + ma - mb) * (M - ma + mb);
  if (!(rad > 0.0)) return 0.0;
  return sqrt(rad) / (2.0 * M);
}
/* O-9: same, with the excess mass M - ma - mb supplied directly (no cancellation).       */
double orc_breakup_excess(double excess, double M, double ma, double mb) {
  double rad = excess * (M + ma + mb) * (M + ma - mb) * (M - ma + mb);
  if (!(rad > 0.0)) return 0.0;
  return sqrt(rad) / (2.0 * M);
}

/* ------------------------------------------------------------------------------------ */
/* O-3 tensors, all with upper (contravariant) indices.                                   */
static const double G4[4] = {1.0, -1.0, -1.0, -1.0};

double orc_dot(const double a[4], const double b[4]) {
  double s = 0.0;
  for (int mu = 0; mu < 4; ++mu) s += a[mu] * G4[mu] * b[mu];
  return s;
}
/* Ptilde^{mu nu}(p) = g^{mu nu} - p^mu p^nu / p^2 */
void orc_proj(const double p[4], double P[4][4]) {
  double p2 = orc_dot(p, p);
  for (int mu = 0; mu < 4; ++mu)
    for (int nu = 0; nu < 4; ++nu) P[mu][nu] = (mu == nu ? G4[mu] : 0.0) - p[mu] * p[nu] / p2;
}
/* L1^mu(p,q) = Ptilde^{mu nu}(p) q_nu  ( = q^mu - p^mu (p.q)/p^2 ) */
void orc_L1(const double p[4], const double q[4], double out[4]) {
  double P[4][4];
  orc_proj(p, P);
  for (int mu = 0; mu < 4; ++mu) {
    double s = 0.0;
    for (int nu = 0; nu < 4; ++nu) s += P[mu][nu] * G4[nu] * q[nu];
    out[mu] = s;
  }
}
/* L2^{mu nu}(p,q) = L1^mu L1^nu - (1/3)(L1.L1) Ptilde^{mu nu}(p) */
void orc_L2(const double p[4], const double q[4], double out[4][4]) {
  double P[4][4], l[4];
  orc_proj(p, P);
  orc_L1(p, q, l);
  double ll = orc_dot(l, l);
  for (int mu = 0; mu < 4; ++mu)
    for (int nu = 0; nu < 4; ++nu) out[mu][nu] = l[mu] * l[nu] - ll * P[mu][nu] / 3.0;
}
/* totally antisymmetric symbol with eps_{0123} = +1: sign of the permutation (a b c d)   */
static int levi(int a, int b, int c, int d) {
  int v[4] = {a, b, c, d};
  if (a == b || a == c || a == d || b == c || b == d || c == d) return 0;
  int sign = 1;
  for (int i = 0; i < 4; ++i)
    for (int j = i + 1; j < 4; ++j)
      if (v[i] > v[j]) sign = -sign;
  return sign;
}
/* eps4(a,b,c,d) = eps_{mu nu rho sigma} a^mu b^nu c^rho d^sigma */
double orc_eps4(const double a[4], const double b[4], const double c[4], const double d[4]) {
  double s = 0.0;
  for (int mu = 0; mu < 4; ++mu)
    for (int nu = 0; nu < 4; ++nu)
      for (int rho = 0; rho < 4; ++rho)
        for (int sg = 0; sg < 4; ++sg) {
          int e = levi(mu, nu, rho, sg);
          if (e) s += e * a[mu] * b[nu] * c[rho] * d[sg];
        }
  return s;
}

/* ------------------------------------------------------------------------------------ */
/* helpers on one event held as p[particle][component]                                    */
static void role_vectors(const int perm[4], const double p[4][4], double r[4][4]) {
  for (int i = 0; i < 4; ++i)
    for (int mu = 0; mu < 4; ++mu) r[i][mu] = p[perm[i]][mu];
}
static void add4(const double a[4], const double b[4], double o[4]) { for (int i = 0; i < 4; ++i) o[i] = a[i] + b[i]; }
static void sub4(const double a[4], const double b[4], double o[4]) { for (int i = 0; i < 4; ++i) o[i] = a[i] - b[i]; }

/* O-4: spin factors (all real), index-loop definitions.  Two topologies:        */
/*   VV kinds : D -> R1 R2, R1 -> r0 r1, R2 -> r2 r3                                       */
/*   cascade  : D -> X r3, X -> V r2, V -> r0 r1                                           */
double orc_spin_factor_event(int sf, const int perm[4], const double p[4][4]) {
  double r[4][4];
  role_vectors(perm, p, r);
  if (sf == ORC_SF_NONRES) return 1.0;
  if (sf == ORC_SF_VV_S || sf == ORC_SF_VV_P || sf == ORC_SF_VV_D) {
    double p1[4], q1[4], p2[4], q2[4], pD[4], qD[4], v1[4], v2[4];
    add4(r[0], r[1], p1); sub4(r[0], r[1], q1);
    add4(r[2], r[3], p2); sub4(r[2], r[3], q2);
    add4(p1, p2, pD);     sub4(p1, p2, qD);
    orc_L1(p1, q1, v1);
    orc_L1(p2, q2, v2);
    if (sf == ORC_SF_VV_S) return orc_dot(v1, v2);                 /* v1^mu v2_mu            */
    if (sf == ORC_SF_VV_P) return orc_eps4(pD, qD, v1, v2);        /* eps(pD, qD, v1, v2)    */
    double L2D[4][4], s = 0.0;                                     /* L2^{mu nu} v1_mu v2_nu */
    orc_L2(pD, qD, L2D);
    for (int mu = 0; mu < 4; ++mu)
      for (int nu = 0; nu < 4; ++nu) s += L2D[mu][nu] * (G4[mu] * v1[mu]) * (G4[nu] * v2[nu]);
    return s;
  }
  /* cascade kinds */
  double pV[4], qV[4], pX[4], qX[4], pD[4], qD[4], v[4], d[4];
  add4(r[0], r[1], pV); sub4(r[0], r[1], qV);
  add4(pV, r[2], pX);   sub4(pV, r[2], qX);
  add4(pX, r[3], pD);   sub4(pX, r[3], qD);
  orc_L1(pV, qV, v);
  orc_L1(pD, qD, d);
  if (sf == ORC_SF_AP_S) {                                         /* -d_mu Pt^{mu nu}(pX) v_nu */
    double P[4][4], s = 0.0;
    orc_proj(pX, P);
    for (int mu = 0; mu < 4; ++mu)
      for (int nu = 0; nu < 4; ++nu) s += (G4[mu] * d[mu]) * P[mu][nu] * (G4[nu] * v[nu]);
    return -s;
  }
  if (sf == ORC_SF_AP_D) {                                         /* d_mu L2^{mu nu}(pX,qX) v_nu: axial -> V P in D-wave */
    double L2X[4][4], s = 0.0;
    orc_L2(pX, qX, L2X);
    for (int mu = 0; mu < 4; ++mu)
      for (int nu = 0; nu < 4; ++nu) s += (G4[mu] * d[mu]) * L2X[mu][nu] * (G4[nu] * v[nu]);
    return s;
  }
  if (sf == ORC_SF_TP_D) {
    /* L2^{rho sg}(pD,qD) eps_{rho al be ga} L2(pX,qX)_sg^al pX^be v^ga */
    double L2D[4][4], L2T[4][4], s = 0.0;
    orc_L2(pD, qD, L2D);
    orc_L2(pX, qX, L2T);
    for (int rho = 0; rho < 4; ++rho)
      for (int sg = 0; sg < 4; ++sg)
        for (int al = 0; al < 4; ++al)
          for (int be = 0; be < 4; ++be)
            for (int ga = 0; ga < 4; ++ga) {
              int e = levi(rho, al, be, ga);
              if (e) s += L2D[rho][sg] * e * (G4[sg] * L2T[sg][al]) * pX[be] * v[ga];
            }
    return s;
  }
  return NAN;
}

/* O-5: un-normalised Blatt-Weisskopf factors, z = (q r)^2 */
double orc_barrier(int L, double z) {
  if (L == 0) return 1.0;
  if (L == 1) return 1.0 / sqrt(1.0 + z);
  if (L == 2) return 1.0 / sqrt(9.0 + 3.0 * z + z * z);
  return NAN;
}

/* O-6: relativistic Breit-Wigner with mass-dependent width.                              */
/*   T(s) = 1 / (m0^2 - s - i m0 Gamma(s)),                                                */
/*   Gamma(s) = Gamma0 (q/q0)^{2L+1} (m0/sqrt s) [F_L(z)/F_L(z0)]^2.                       */
/* (ma, mb): daughter masses at s (running); (ma0, mb0): at the pole.  Returns 0, or -1 on */
/* a domain error (pole below its own threshold).                                         */
int orc_breit_wigner(double m0, double gamma0, int L, double r, double s, double ma, double mb,
                     double ma0, double mb0, double out[2]) {
  if (!(m0 > ma0 + mb0)) { out[0] = out[1] = NAN; return -1; }
  double m = sqrt(s);
  double q = orc_breakup(m, ma, mb), q0 = orc_breakup(m0, ma0, mb0);
  double z = (q * r) * (q * r), z0 = (q0 * r) * (q0 * r);
  double fr = orc_barrier(L, z) / orc_barrier(L, z0);
  double gamma = gamma0 * pow(q / q0, 2 * L + 1) * (m0 / m) * fr * fr;
  double complex T = 1.0 / ((m0 * m0 - s) - I * (m0 * gamma));
  out[0] = creal(T); out[1] = cimag(T);
  return 0;
}

/* Breit-Wigner with constant width (lineshape kind 1): T(s) = 1 / (m0^2 - s - i m0 Gamma0).  No threshold enters. */
void orc_breit_wigner_constant(double m0, double gamma0, double s, double out[2]) {
  double complex T = 1.0 / ((m0 * m0 - s) - I * (m0 * gamma0));
  out[0] = creal(T); out[1] = cimag(T);
}

/* L of the D vertex for each spin-factor kind (O-5) */
static int parent_L(int sf) {
  switch (sf) {
    case ORC_SF_VV_S: return 0; case ORC_SF_VV_P: return 1; case ORC_SF_VV_D: return 2;
    case ORC_SF_AP_S: return 1; case ORC_SF_TP_D: return 2; case ORC_SF_AP_D: return 1; default: return 0;
  }
}
/* radius of resonance R's own decay vertex, and its lineshape by kind */
static double res_radius(const orc_model *m, int R) { return m->res_r[R] > 0.0 ? m->res_r[R] : m->r_res; }
static int lineshape(const orc_model *m, const orc_params *par, int R, double s, double ma, double mb, double ma0,
                     double mb0, double out[2]) {
  if (m->res_kind[R] == ORC_LS_CONSTANT) { orc_breit_wigner_constant(par->mass[R], par->width[R], s, out); return 0; }
  return orc_breit_wigner(par->mass[R], par->width[R], m->res_L[R], res_radius(m, R), s, ma, mb, ma0, mb0, out);
}

/* O-2: one decay-chain amplitude a_k = S_k F_{L_D}(z_D) prod_R [F_{L_R}(z_R) T_R]. */
/* parts (may be NULL): [0] S_k, [1] product of all barrier factors, [2..3] product of T_R. */
int orc_term_event(const orc_model *m, const orc_params *par, int k, const double p[4][4],
                   double out[2], double parts[4]) {
  int sf = m->term_sf[k];
  const int *perm = m->term_perm[k];
  double S = orc_spin_factor_event(sf, perm, p);
  double F = 1.0;
  double complex T = 1.0;
  int status = 0;
  if (sf != ORC_SF_NONRES) {
    double r[4][4], pD[4] = {0, 0, 0, 0};
    role_vectors(perm, p, r);
    for (int i = 0; i < 4; ++i) add4(pD, r[i], pD);
    double mD = sqrt(orc_dot(pD, pD));
    int R0 = m->term_res[k][0], R1 = m->term_res[k][1];
    double bw[2];
    if (sf == ORC_SF_VV_S || sf == ORC_SF_VV_P || sf == ORC_SF_VV_D) {
      double p1[4], p2[4];
      add4(r[0], r[1], p1); add4(r[2], r[3], p2);
      double s1 = orc_dot(p1, p1), s2 = orc_dot(p2, p2);
      double ma = m->m_final[perm[0]], mb = m->m_final[perm[1]];
      double mc = m->m_final[perm[2]], md = m->m_final[perm[3]];
      double qD = orc_breakup(mD, sqrt(s1), sqrt(s2));
      double q1 = orc_breakup(sqrt(s1), ma, mb), q2 = orc_breakup(sqrt(s2), mc, md);
      F *= orc_barrier(parent_L(sf), (qD * m->r_parent) * (qD * m->r_parent));
      F *= orc_barrier(m->res_L[R0], (q1 * res_radius(m, R0)) * (q1 * res_radius(m, R0)));
      F *= orc_barrier(m->res_L[R1], (q2 * res_radius(m, R1)) * (q2 * res_radius(m, R1)));
      status |= lineshape(m, par, R0, s1, ma, mb, ma, mb, bw);
      T *= bw[0] + I * bw[1];
      status |= lineshape(m, par, R1, s2, mc, md, mc, md, bw);
      T *= bw[0] + I * bw[1];
    } else {
      double pV[4], pX[4];
      add4(r[0], r[1], pV); add4(pV, r[2], pX);
      double sV = orc_dot(pV, pV), sX = orc_dot(pX, pX);
      double ma = m->m_final[perm[0]], mb = m->m_final[perm[1]];
      double mc = m->m_final[perm[2]], md = m->m_final[perm[3]];
      double qD = orc_breakup(mD, sqrt(sX), md);
      double qX = orc_breakup(sqrt(sX), sqrt(sV), mc);
      double qV = orc_breakup(sqrt(sV), ma, mb);
      F *= orc_barrier(parent_L(sf), (qD * m->r_parent) * (qD * m->r_parent));
      F *= orc_barrier(m->res_L[R0], (qX * res_radius(m, R0)) * (qX * res_radius(m, R0)));
      F *= orc_barrier(m->res_L[R1], (qV * res_radius(m, R1)) * (qV * res_radius(m, R1)));
      /* X -> V c: running daughter mass at s, the daughter's current m0 at the pole (O-6) */
      status |= lineshape(m, par, R0, sX, sqrt(sV), mc, par->mass[R1], mc, bw);
      T *= bw[0] + I * bw[1];
      status |= lineshape(m, par, R1, sV, ma, mb, ma, mb, bw);
      T *= bw[0] + I * bw[1];
    }
  }
  double complex a = S * F * T;
  out[0] = creal(a); out[1] = cimag(a);
  if (parts) { parts[0] = S; parts[1] = F; parts[2] = creal(T); parts[3] = cimag(T); }
  return status;
}

/* eq. (2): A_f = sum_k c_kappa(k) a_k, Abar_f = sum_k cbar_kappa(k) a_k.         */
int orc_amplitudes_event(const orc_model *m, const orc_params *par, const double p[4][4],
                         double A[2], double Abar[2]) {
  double complex a = 0.0, ab = 0.0;
  int status = 0;
  for (int k = 0; k < m->n_terms; ++k) {
    double ak[2];
    status |= orc_term_event(m, par, k, p, ak, NULL);
    int kap = m->term_coupling[k];
    double complex z = ak[0] + I * ak[1];
    a += (par->c[kap][0] + I * par->c[kap][1]) * z;
    ab += (par->cbar[kap][0] + I * par->cbar[kap][1]) * z;
  }
  A[0] = creal(a); A[1] = cimag(a); Abar[0] = creal(ab); Abar[1] = cimag(ab);
  return status;
}

/* eq. (1): the bracket B; R = e^{-Gamma t} B, Gamma = 1/tau (O-1).               */
double orc_bracket(const double A[2], const double Abar[2], double x, double y, double Gamma, double t) {
  double complex a = A[0] + I * A[1], ab = Abar[0] + I * Abar[1];
  double aa = creal(a * conj(a)), bb = creal(ab * conj(ab));
  double complex cross = a * conj(ab);
  return (aa + bb) * cosh(y * Gamma * t) + (aa - bb) * cos(x * Gamma * t)
         - 2.0 * creal(cross) * sinh(y * Gamma * t) - 2.0 * cimag(cross) * sin(x * Gamma * t);
}

/* O-8 (no resolution): integrals over [t_lo, t_hi] of e^{-Gamma t}{cosh, cos, sinh, sin}. */
/* I(lambda) = (e^{-lambda t_lo} - e^{-lambda t_hi}) / lambda;                              */
/* cosh -> [I(l-) + I(l+)]/2, sinh -> [I(l-) - I(l+)]/2, l-+ = Gamma(1 -+ y);               */
/* cos -> Re I(lx), sin -> Im I(lx), lx = Gamma(1 - i x).                                   */
static double complex window_integral(double complex lambda, double t_lo, double t_hi) {
  double complex lo = cexp(-lambda * t_lo);
  double complex hi = isinf(t_hi) ? 0.0 : cexp(-lambda * t_hi);
  return (lo - hi) / lambda;
}
void orc_time_integrals(double x, double y, double tau, double t_lo, double t_hi, double T[4]) {
  double Gamma = 1.0 / tau;
  double complex Im = window_integral(Gamma * (1.0 - y), t_lo, t_hi);
  double complex Ip = window_integral(Gamma * (1.0 + y), t_lo, t_hi);
  double complex Ix = window_integral(Gamma * (1.0 - I * x), t_lo, t_hi);
  T[0] = 0.5 * (creal(Im) + creal(Ip));
  T[1] = creal(Ix);
  T[2] = 0.5 * (creal(Im) - creal(Ip));
  T[3] = cimag(Ix);
}

/* ------------------------------------------------------------------------------------ */
/* batch entry points (SoA in, one slot per event out)                                    */
static void load_event(const double *p4, int64_t n, int64_t i, double p[4][4]) {
  for (int a = 0; a < 4; ++a)
    for (int mu = 0; mu < 4; ++mu) p[a][mu] = p4[(int64_t)(4 * a + mu) * n + i];
}

/* per-term pieces for per-layer parity: S[k][n], F[k][n] (barrier product), a[k][n][2]   */
int orc_terms(const orc_model *m, const orc_params *par, int64_t n, const double *p4,
              double *S, double *F, double *a) {
  int status = 0;
#pragma omp parallel for schedule(static) reduction(| : status)
  for (int64_t i = 0; i < n; ++i) {
    double p[4][4];
    load_event(p4, n, i, p);
    for (int k = 0; k < m->n_terms; ++k) {
      double ak[2], parts[4];
      status |= orc_term_event(m, par, k, p, ak, parts);
      if (S) S[(int64_t)k * n + i] = parts[0];
      if (F) F[(int64_t)k * n + i] = parts[1];
      if (a) { a[((int64_t)k * n + i) * 2] = ak[0]; a[((int64_t)k * n + i) * 2 + 1] = ak[1]; }
    }
  }
  return status;
}

/* A[n][2], Abar[n][2] */
int orc_amplitudes(const orc_model *m, const orc_params *par, int64_t n, const double *p4,
                   double *A, double *Abar) {
  int status = 0;
#pragma omp parallel for schedule(static) reduction(| : status)
  for (int64_t i = 0; i < n; ++i) {
    double p[4][4];
    load_event(p4, n, i, p);
    status |= orc_amplitudes_event(m, par, p, A + 2 * i, Abar + 2 * i);
  }
  return status;
}

/* step 6 / O-8: N = (1/N_n) sum_j w_j int R(p_j, t) dt over the normalisation sample      */
/* (P:55), direct sum; also returns S_1..S_4 (may be NULL).                                */
int orc_norm(const orc_model *m, const orc_params *par, int64_t n, const double *p4, const double *w,
             double *norm_out, double S_out[4]) {
  double *A = malloc(sizeof(double) * 2 * n), *Ab = malloc(sizeof(double) * 2 * n);
  int status = orc_amplitudes(m, par, n, p4, A, Ab);
  double T[4];
  orc_time_integrals(par->x, par->y, par->tau, m->t_lo, m->t_hi, T);
  orc_acc tot = {0, 0}, s1 = {0, 0}, s2 = {0, 0}, s3 = {0, 0}, s4 = {0, 0};
  for (int64_t j = 0; j < n; ++j) {
    double complex a = A[2 * j] + I * A[2 * j + 1], ab = Ab[2 * j] + I * Ab[2 * j + 1];
    double aa = creal(a * conj(a)), bb = creal(ab * conj(ab));
    double complex cross = a * conj(ab);
    double wj = w ? w[j] : 1.0;
    acc_add(&tot, wj * (T[0] * (aa + bb) + T[1] * (aa - bb) - 2.0 * T[2] * creal(cross) - 2.0 * T[3] * cimag(cross)));
    acc_add(&s1, wj * (aa + bb)); acc_add(&s2, wj * (aa - bb));
    acc_add(&s3, wj * creal(cross)); acc_add(&s4, wj * cimag(cross));
  }
  *norm_out = acc_value(&tot) / (double)n;          /* 1/N_n, not 1/sum w (O-8) */
  if (S_out) {
    S_out[0] = acc_value(&s1) / (double)n; S_out[1] = acc_value(&s2) / (double)n;
    S_out[2] = acc_value(&s3) / (double)n; S_out[3] = acc_value(&s4) / (double)n;
  }
  free(A); free(Ab);
  return status;
}

/* unnormalised rate R_i = e^{-Gamma t_i} B_i and bracket B_i per event (either may be NULL) */
int orc_rate(const orc_model *m, const orc_params *par, int64_t n, const double *p4, const double *t,
             double *R, double *B) {
  int status = 0;
  double Gamma = 1.0 / par->tau;
#pragma omp parallel for schedule(static) reduction(| : status)
  for (int64_t i = 0; i < n; ++i) {
    double p[4][4], A[2], Ab[2];
    load_event(p4, n, i, p);
    status |= orc_amplitudes_event(m, par, p, A, Ab);
    double b = orc_bracket(A, Ab, par->x, par->y, Gamma, t[i]);
    if (B) B[i] = b;
    if (R) R[i] = exp(-Gamma * t[i]) * b;
  }
  return status;
}

/* step 7: P_i = R_i / N and NLL = -sum_i log P_i (O-8).  prob may be NULL.     */
/* Returns 0; 1 if a resonance pole is below threshold; 2 if some P_i <= 0 or non-finite    */
/* (then *nll_out = +inf).                                                                  */
int orc_nll(const orc_model *m, const orc_params *par, int64_t n, const double *p4, const double *t,
            int64_t n_norm, const double *p4_norm, const double *w_norm,
            double *nll_out, double *norm_out, double *prob) {
  double norm;
  int status = orc_norm(m, par, n_norm, p4_norm, w_norm, &norm, NULL);
  double *R = malloc(sizeof(double) * n);
  status |= orc_rate(m, par, n, p4, t, R, NULL);
  orc_acc acc = {0, 0};
  int bad = 0;
  for (int64_t i = 0; i < n; ++i) {
    double P = R[i] / norm;
    if (prob) prob[i] = P;
    if (!(P > 0.0) || !isfinite(P)) bad = 1; else acc_add(&acc, log(P));
  }
  free(R);
  if (norm_out) *norm_out = norm;
  *nll_out = bad ? INFINITY : -acc_value(&acc);
  return status ? 1 : (bad ? 2 : 0);
}

/* ------------------------------------------------------------------------------------ */
/* O-9 / G2-G3: one Raubold-Lynch candidate.  Blocks: 0 (r, r'), 1..3 (cos theta, phi) of   */
/* decays D->X3+[3], X3->X2+[2], X2->[0]+[1]; 4 (u_t, u_acc).                               */
static void boost(const double P[4], double M, const double p[4], double out[4]) {
  /* E' = (E_P E + P.p)/M;  p' = p + P [ (P.p)/(M (E_P + M)) + E/M ]  (O-9) */
  double Pp = P[1] * p[1] + P[2] * p[2] + P[3] * p[3];
  double f = Pp / (M * (P[0] + M)) + p[0] / M;
  out[0] = (P[0] * p[0] + Pp) / M;
  for (int i = 1; i < 4; ++i) out[i] = p[i] + P[i] * f;
}
static void two_body(double M, double m_first, double m_second, double pstar, double u_cos, double u_phi,
                     double first[4], double second[4]) {
  double ct = 2.0 * u_cos - 1.0, phi = 2.0 * M_PI * u_phi;
  double st = sqrt(1.0 - ct * ct);
  double nx = st * cos(phi), ny = st * sin(phi), nz = ct;
  (void)M;
  first[0] = sqrt(m_first * m_first + pstar * pstar);
  first[1] = pstar * nx; first[2] = pstar * ny; first[3] = pstar * nz;
  second[0] = sqrt(m_second * m_second + pstar * pstar);
  second[1] = -pstar * nx; second[2] = -pstar * ny; second[3] = -pstar * nz;
}
void orc_candidate(const orc_model *m, double tau, uint64_t seed, uint32_t stream, uint64_t i,
                   double p[4][4], double *t, double *w, double *u_acc) {
  double ur[2], u1[2], u2[2], u3[2], ut[2];
  orc_uniform_pair(seed, i, 0, stream, ur);
  orc_uniform_pair(seed, i, 1, stream, u1);
  orc_uniform_pair(seed, i, 2, stream, u2);
  orc_uniform_pair(seed, i, 3, stream, u3);
  orc_uniform_pair(seed, i, 4, stream, ut);
  const double *mf = m->m_final;
  double r1 = ur[0] < ur[1] ? ur[0] : ur[1], r2 = ur[0] < ur[1] ? ur[1] : ur[0];
  double Tk = m->m_parent - (mf[0] + mf[1] + mf[2] + mf[3]);
  double M2 = mf[0] + mf[1] + r1 * Tk, M3 = mf[0] + mf[1] + mf[2] + r2 * Tk, M4 = m->m_parent;
  double ps1 = orc_breakup_excess((1.0 - r2) * Tk, M4, M3, mf[3]);
  double ps2 = orc_breakup_excess((r2 - r1) * Tk, M3, M2, mf[2]);
  double ps3 = orc_breakup_excess(r1 * Tk, M2, mf[0], mf[1]);
  double X3[4], X2[4], a[4], b[4], tmp[4];
  two_body(M4, M3, mf[3], ps1, u1[0], u1[1], X3, p[3]);          /* D rest frame            */
  two_body(M3, M2, mf[2], ps2, u2[0], u2[1], X2, tmp);           /* X3 rest frame           */
  boost(X3, M3, tmp, p[2]);
  two_body(M2, mf[0], mf[1], ps3, u3[0], u3[1], a, b);           /* X2 rest frame           */
  boost(X2, M2, a, tmp); boost(X3, M3, tmp, p[0]);
  boost(X2, M2, b, tmp); boost(X3, M3, tmp, p[1]);
  *w = ps1 * ps2 * ps3;
  *t = -tau * log(1.0 - ut[0]);
  *u_acc = ut[1];
}

/* candidates first .. first+n-1: p4[16][n] SoA, t[n], w[n], u_acc[n] (any may be NULL)     */
void orc_candidates(const orc_model *m, double tau, uint64_t seed, uint32_t stream, uint64_t first, int64_t n,
                    double *p4, double *t, double *w, double *u_acc) {
#pragma omp parallel for schedule(static)
  for (int64_t j = 0; j < n; ++j) {
    double p[4][4], tj, wj, uj;
    orc_candidate(m, tau, seed, stream, first + (uint64_t)j, p, &tj, &wj, &uj);
    if (p4)
      for (int a = 0; a < 4; ++a)
        for (int mu = 0; mu < 4; ++mu) p4[(int64_t)(4 * a + mu) * n + j] = p[a][mu];
    if (t) t[j] = tj;
    if (w) w[j] = wj;
    if (u_acc) u_acc[j] = uj;
  }
}

/* same for an explicit list of candidate indices (full-size parity: the oracle regenerates the  */
/* events itself from (seed, index) instead of being handed momenta)                            */
void orc_candidates_at(const orc_model *m, double tau, uint64_t seed, uint32_t stream, int64_t n,
                       const int64_t *index, double *p4, double *t, double *w, double *u_acc) {
#pragma omp parallel for schedule(static)
  for (int64_t j = 0; j < n; ++j) {
    double p[4][4], tj, wj, uj;
    orc_candidate(m, tau, seed, stream, (uint64_t)index[j], p, &tj, &wj, &uj);
    if (p4)
      for (int a = 0; a < 4; ++a)
        for (int mu = 0; mu < 4; ++mu) p4[(int64_t)(4 * a + mu) * n + j] = p[a][mu];
    if (t) t[j] = tj;
    if (w) w[j] = wj;
    if (u_acc) u_acc[j] = uj;
  }
}

/* O-9 / G4: ratio rho_i = w_i B(p_i, t_i) for candidates first .. first+n-1                */
int orc_candidate_ratio(const orc_model *m, const orc_params *par, uint64_t seed, uint32_t stream,
                        uint64_t first, int64_t n, double *rho, double *u_acc) {
  int status = 0;
  double Gamma = 1.0 / par->tau;
#pragma omp parallel for schedule(static) reduction(| : status)
  for (int64_t j = 0; j < n; ++j) {
    double p[4][4], tj, wj, uj, A[2], Ab[2];
    orc_candidate(m, par->tau, seed, stream, first + (uint64_t)j, p, &tj, &wj, &uj);
    status |= orc_amplitudes_event(m, par, p, A, Ab);
    rho[j] = wj * orc_bracket(A, Ab, par->x, par->y, Gamma, tj);
    if (u_acc) u_acc[j] = uj;
  }
  return status;
}

/* O-9 / G5-G6: envelope E = scale * max_{i < n_pilot} rho_i (n_pilot = 0: E = scale);       */
/* accept iff u_acc E < rho; rho > E is accepted and counted as overflow; accepted events    */
/* are written in candidate order.  out_p4 is [16][capacity] SoA.  Returns 0, 1 (pole below  */
/* threshold) or 3 (capacity exceeded; counts are still exact, outputs truncated).          */
int orc_generate(const orc_model *m, const orc_params *par, uint64_t seed, uint32_t stream,
                 int64_t n_candidates, int64_t n_pilot, double envelope_scale, int64_t capacity,
                 double *out_p4, double *out_t, int64_t *out_index,
                 int64_t *n_accepted, int64_t *n_overflow, double *envelope_out) {
  int status = 0;
  double E = envelope_scale;
  const int64_t chunk = 1 << 16;
  double *rho = malloc(sizeof(double) * chunk), *ua = malloc(sizeof(double) * chunk);
  if (n_pilot > 0) {
    double mx = 0.0;
    for (int64_t f = 0; f < n_pilot; f += chunk) {
      int64_t c = n_pilot - f < chunk ? n_pilot - f : chunk;
      status |= orc_candidate_ratio(m, par, seed, stream, (uint64_t)f, c, rho, NULL);
      for (int64_t j = 0; j < c; ++j) if (rho[j] > mx) mx = rho[j];
    }
    E = envelope_scale * mx;
  }
  int64_t nacc = 0, nover = 0;
  for (int64_t f = 0; f < n_candidates; f += chunk) {
    int64_t c = n_candidates - f < chunk ? n_candidates - f : chunk;
    status |= orc_candidate_ratio(m, par, seed, stream, (uint64_t)f, c, rho, ua);
    for (int64_t j = 0; j < c; ++j) {
      if (ua[j] * E < rho[j]) {
        if (rho[j] > E) ++nover;
        if (nacc < capacity) {
          double p[4][4], tj, wj, uj;
          orc_candidate(m, par->tau, seed, stream, (uint64_t)(f + j), p, &tj, &wj, &uj);
          if (out_p4)
            for (int a = 0; a < 4; ++a)
              for (int mu = 0; mu < 4; ++mu) out_p4[(int64_t)(4 * a + mu) * capacity + nacc] = p[a][mu];
          if (out_t) out_t[nacc] = tj;
          if (out_index) out_index[nacc] = f + j;
        }
        ++nacc;
      }
    }
  }
  free(rho); free(ua);
  *n_accepted = nacc; *n_overflow = nover; *envelope_out = E;
  if (status) return 1;
  return nacc > capacity ? 3 : 0;
}

/* single-event spin factor from a flat [4][4] array (for the pins) */
double orc_spin_factor(int sf, const int perm[4], const double *p16) {
  double p[4][4];
  memcpy(p, p16, sizeof(p));
  return orc_spin_factor_event(sf, perm, p);
}
