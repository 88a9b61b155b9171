"""Independent numpy helpers for the oracle pins (Lorentz boosts, closed-form spin factors).
They restate nothing from oracle/: closed forms and rest-frame reductions are a different route to
the same numbers than the oracle's explicit index loops."""
import numpy as np

G = np.diag([1.0, -1.0, -1.0, -1.0])


def dot(a, b):
    return a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3]


def boost_matrix(beta):
    """Lorentz boost with velocity vector beta (|beta| < 1): rest-frame vector -> moving frame."""
    beta = np.asarray(beta, float)
    b2 = beta @ beta
    g = 1.0 / np.sqrt(1.0 - b2)
    L = np.eye(4)
    L[0, 0] = g
    L[0, 1:] = g * beta
    L[1:, 0] = g * beta
    if b2 > 0:
        L[1:, 1:] += (g - 1.0) * np.outer(beta, beta) / b2
    return L


def boost_to_rest(p):
    """Matrix taking vectors into the rest frame of four-momentum p."""
    return boost_matrix(-np.asarray(p[1:]) / p[0])


def rotation(rng):
    q, r = np.linalg.qr(rng.standard_normal((3, 3)))
    q = q * np.sign(np.diag(r))
    if np.linalg.det(q) < 0:
        q[:, 0] = -q[:, 0]
    R = np.eye(4)
    R[1:, 1:] = q
    return R


def L1(p, q):
    return q - p * dot(p, q) / dot(p, p)


def eps4(a, b, c, d):
    return np.linalg.det(np.stack([a, b, c, d], axis=1))


def breakup(M, a, b):
    rad = (M - a - b) * (M + a + b) * (M + a - b) * (M - a + b)
    return np.sqrt(max(rad, 0.0)) / (2 * M)


def closed_spin_factor(sf, perm, p):
    """Closed forms of O-4 (right-hand sides), p[particle][component] of one event."""
    r = [np.asarray(p[perm[i]], float) for i in range(4)]
    if sf == 0:
        return 1.0
    if sf in (1, 2, 3):
        p1, q1, p2, q2 = r[0] + r[1], r[0] - r[1], r[2] + r[3], r[2] - r[3]
        pD, qD = p1 + p2, p1 - p2
        v1, v2, d = L1(p1, q1), L1(p2, q2), L1(pD, qD)
        if sf == 1:
            return dot(v1, v2)
        if sf == 2:
            return eps4(pD, qD, v1, v2)
        mD2 = dot(pD, pD)
        return dot(d, v1) * dot(d, v2) - dot(d, d) / 3.0 * (dot(v1, v2) - dot(pD, v1) * dot(pD, v2) / mD2)
    pV, qV = r[0] + r[1], r[0] - r[1]
    pX, qX = pV + r[2], pV - r[2]
    pD, qD = pX + r[3], pX - r[3]
    v, d, t = L1(pV, qV), L1(pD, qD), L1(pX, qX)
    if sf == 4:
        return -(dot(d, v) - dot(pX, d) * dot(pX, v) / dot(pX, pX))
    if sf == 5:
        mD2 = dot(pD, pD)
        return dot(d, t) * eps4(d, t, pX, v) + dot(d, d) / 3.0 * dot(pD, t) / mD2 * eps4(pD, t, pX, v)
    if sf == 6:     # d_mu L2^{mu nu}(pX, qX) v_nu = (d.t)(t.v) - (t.t)/3 [d.v - (pX.d)(pX.v)/sX]
        return dot(d, t) * dot(t, v) - dot(t, t) / 3.0 * (dot(d, v) - dot(pX, d) * dot(pX, v) / dot(pX, pX))
    raise ValueError(sf)


def event(p4, i):
    """[16][n] SoA -> [4][4] of event i."""
    return np.asarray(p4)[:, i].reshape(4, 4)
