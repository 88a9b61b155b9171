"""Validation observables of the paper's Fig. 3 ("projections ... m12, m34, cos12, cos34, phi").
TEST INFRASTRUCTURE, NOT THE PRODUCT.

The paper names the five observables and does not define them.  Reading ("standard
helicity angles"), with the final state ordered 0 = K+, 1 = pi-, 2 = pi+, 3 = pi- and the pairing 12 = (pi+ pi-) =
particles (2, 3), 34 = (K+ pi-) = particles (0, 1):

  m12, m34   invariant masses of the two pairs;
  cos12      cosine of the angle between the pi+ momentum in the (2,3) rest frame and the flight direction of the (2,3)
             system in the D rest frame (helicity angle);
  cos34      the same for the K+ in the (0,1) rest frame and the flight direction of the (0,1) system;
  phi        angle between the two decay planes in the D rest frame: with z = unit vector along the (2,3) system,
             n12 = p2 x p3 / |p2 x p3|, n34 = p0 x p1 / |p0 x p1|:  cos phi = n12 . n34,  sin phi = (n12 x n34) . z,
             phi = atan2(sin phi, cos phi) in (-pi, pi].

Written as the definitions say: explicit Lorentz boosts into the D, (2,3) and (0,1) rest frames, three-vector dot and
cross products, numpy only.  Pins (tests/test_oracle_projections.py): Lorentz invariance under random boosts and
rotations; the invariant (boost-free) closed form of a helicity cosine; parity (phi -> -phi) and pi+ <-> pi- exchange
(cos12 -> -cos12); flat phase space gives flat cos12, cos34 and phi; a planar event has phi in {0, pi}.
"""
from __future__ import annotations

import numpy as np

NAMES = ("m12", "m34", "cos12", "cos34", "phi")
PAIR12 = (2, 3)     # pi+ pi-
PAIR34 = (0, 1)     # K+ pi-


def _vec(p4, a):
    """Four-momentum of particle a: [4][n] (E, px, py, pz) from the SoA [16][n]."""
    return np.asarray(p4, dtype=np.float64)[4 * a:4 * a + 4]


def _mass2(p):
    return p[0] * p[0] - p[1] * p[1] - p[2] * p[2] - p[3] * p[3]


def boost_to_rest_frame_of(P, p):
    """p seen from the rest frame of P (both [4][n]): the standard boost with velocity -P_vec / P_E."""
    M = np.sqrt(_mass2(P))
    Pp = P[1] * p[1] + P[2] * p[2] + P[3] * p[3]
    E = (P[0] * p[0] - Pp) / M
    f = (Pp / (P[0] + M) - p[0]) / M
    return np.stack([E, p[1] + f * P[1], p[2] + f * P[2], p[3] + f * P[3]])


def _unit(v):
    return v / np.sqrt(np.sum(v * v, axis=0))


def observables(p4):
    """[5][n]: m12, m34, cos12, cos34, phi of every event."""
    p = [_vec(p4, a) for a in range(4)]
    D = p[0] + p[1] + p[2] + p[3]
    q = [boost_to_rest_frame_of(D, v) for v in p]               # everything in the D rest frame
    P12, P34 = q[PAIR12[0]] + q[PAIR12[1]], q[PAIR34[0]] + q[PAIR34[1]]
    m12, m34 = np.sqrt(_mass2(P12)), np.sqrt(_mass2(P34))
    z12, z34 = _unit(P12[1:]), _unit(P34[1:])                    # flight directions in the D rest frame
    a12 = boost_to_rest_frame_of(P12, q[PAIR12[0]])[1:]          # pi+ in the (2,3) rest frame
    a34 = boost_to_rest_frame_of(P34, q[PAIR34[0]])[1:]          # K+ in the (0,1) rest frame
    cos12 = np.sum(_unit(a12) * z12, axis=0)
    cos34 = np.sum(_unit(a34) * z34, axis=0)
    n12 = _unit(np.cross(q[PAIR12[0]][1:], q[PAIR12[1]][1:], axis=0))
    n34 = _unit(np.cross(q[PAIR34[0]][1:], q[PAIR34[1]][1:], axis=0))
    cphi = np.sum(n12 * n34, axis=0)
    sphi = np.sum(np.cross(n12, n34, axis=0) * z12, axis=0)
    return np.stack([m12, m34, cos12, cos34, np.arctan2(sphi, cphi)])


def default_ranges(m_parent, m_final):
    """[5][2] histogram ranges: the kinematic limits of the two masses, [-1, 1] for the cosines, [-pi, pi] for phi."""
    m = m_final
    return np.array([[m[2] + m[3], m_parent - m[0] - m[1]], [m[0] + m[1], m_parent - m[2] - m[3]],
                     [-1.0, 1.0], [-1.0, 1.0], [-np.pi, np.pi]])


def histograms(p4, n_bins, ranges):
    """Counts [5][n_bins] (int64): bin = floor((v - lo) / (hi - lo) * n_bins), values outside [lo, hi) are dropped,
    v == hi goes to the last bin."""
    obs = observables(p4)
    out = np.zeros((5, n_bins), dtype=np.int64)
    for k in range(5):
        lo, hi = ranges[k]
        b = np.floor((obs[k] - lo) / (hi - lo) * n_bins).astype(np.int64)
        b[obs[k] == hi] = n_bins - 1
        ok = (b >= 0) & (b < n_bins)
        out[k] = np.bincount(b[ok], minlength=n_bins)
    return out
