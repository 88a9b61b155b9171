// tables.h -- plain-data tables handed to the kernels by value (they live in the constant bank).
// Internal to csrc/; the public boundary is include/tddp4.h.
#pragma once
#ifdef __CUDACC_RTC__       // NVRTC has no system headers (this file is also part of run-time compiled programs, jit.h)
typedef signed char int8_t; typedef unsigned char uint8_t; typedef int int32_t; typedef unsigned int uint32_t;
typedef long long int64_t; typedef unsigned long long uint64_t;
#else
#include <stdint.h>
#endif
#include "nll_shared.cuh"

namespace tddp4k {

constexpr int MAX_SYS = 12;    // distinct particle systems (2-, 3- and the 4-body one)
constexpr int MAX_INST = 24;   // de-duplicated lineshape instances
static_assert(MAX_INST == TDDP4_MAX_INST, "jit_shared.cuh");
constexpr int MAX_TERMS = 32;
constexpr int MAX_KC = 16;
static_assert(MAX_KC == TDDP4_MAX_KC, "nll_shared.cuh");
constexpr int MAX_RES = 16;

enum { SF_NONRES = 0, SF_VV_S = 1, SF_VV_P = 2, SF_VV_D = 3, SF_AP_S = 4, SF_TP_D = 5, SF_AP_D = 6 };
enum { LS_RUNNING = 0, LS_CONSTANT = 1 };   // lineshape kinds: mass-dependent width (O-6), constant width

struct InstTab {     // one lineshape instance = (resonance, system it sits on, running daughter)
  int8_t res;        // resonance index
  int8_t sys;        // index of the system whose s is the running mass squared
  int8_t sub;        // system index of the running daughter (cascade X -> V c), -1: two stable daughters
  int8_t L;          // L of the resonance's decay vertex
  int8_t dres;       // daughter resonance (its current m0 enters q0), -1 none
  int8_t kind;       // LS_*: a constant-width instance has the shape g = 1 and gam = m0 Gamma0
  int8_t grow;       // row of its shape g among the g rows of the cache: instances that differ only in the resonance share one
  int8_t pad[1];
  double ma, mb;     // fixed daughter masses (ma unused when sub >= 0)
  double r2;         // Blatt-Weisskopf radius squared of this resonance's own vertex, GeV^-2
};

struct TermTab {     // one decay chain (one Bose ordering)
  int8_t sf;         // spin-factor kind
  int8_t LD;         // L of the D vertex
  int8_t inst0;      // VV: R1; cascade: X.  -1 none
  int8_t inst1;      // VV: R2; cascade: V.  -1 none
  int8_t perm[4];    // role -> particle
  int8_t frow;       // row of its static factor f among the f rows of the cache (shared by chains that differ only in the
                     // resonances); -1: non-resonant term, f = 1, no row
};

struct ModelTab {
  int n_sys, n_inst, n_terms, n_kc;
  int n_g, n_f;                    // distinct shape rows (<= n_inst) and static-factor rows (<= n_terms) of the cache
  int sysD;                        // index of the four-body system
  uint8_t sys_mask[MAX_SYS];
  int n_su;                        // systems whose s some lineshape instance reads (they are numbered last)
  // One three-body system whose s is a combination of streamed s rows is not streamed itself (n_sd = 1; it is numbered just
  // before the streamed ones, so its stored row sits in the part of the tile the per-call kernels skip):
  //   s_{pqy} = s_{pqx} - s_{px} - s_{qx} + s_{py} + s_{qy} + m_x^2 - m_y^2      (the pair pq and its masses cancel), or
  //   s_{abc} = s_{ab} + s_{ac} + s_{bc} - m_a^2 - m_b^2 - m_c^2
  int n_sd;                        // 0 or 1
  int8_t sd_coef[MAX_SYS];         // coefficient (-1, 0, +1) of streamed row r (0 .. n_su-1) in the derived s
  double sd_const;                 // the mass terms
  int8_t col_begin[MAX_KC + 1];    // terms (sorted by coupling) of column kappa: [col_begin[k], col_begin[k+1])
  int8_t user_term[MAX_TERMS];     // sorted position -> caller's term index
  InstTab inst[MAX_INST];
  TermTab term[MAX_TERMS];
  double m_final[4];
  double m_parent;
  double r_res2, r_parent2;        // default resonance radius and parent radius, squared, GeV^-2
};

// The static cache of one event set is ONE tile-major array: tile = 32 consecutive events, R rows of 32 doubles each
// (256 B per row per tile), rows ordered
//   [ s: n_sys | g: n_g | f: n_f | w (if weighted) ]   (n_g, n_f: distinct rows, ModelTab),
// element (row r, event i) at ((i >> 5) * R + r) * 32 + (i & 31).  A warp working on one tile therefore addresses every
// row as tile base + lane + CONSTANT, and the whole tile is one contiguous R * 256-byte region of HBM.  The fused
// per-call kernels get these offsets (and the model tables) as compile-time constants (jit_prelude in tddp4_api.cu).
struct CacheLayout {
  int R;                           // rows per tile of an unweighted event set (+ 1 with weights)
  int g_off, f_off;                // element offsets (row * 32) of the first g row and the first f row
  int skip;                        // element offset of the first row the per-call kernels read (unused s rows come first)
};

}  // namespace tddp4k
