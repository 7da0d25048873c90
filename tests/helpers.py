"""Test-side helpers: explicit Dirac algebra and 2->2 kinematics (numpy only).

Independent of both the oracle and the CUDA path: used to pin the oracle's matrix
elements against explicit traces and textbook closed forms.
"""
import numpy as np

I2 = np.eye(2, dtype=complex)
Z2 = np.zeros((2, 2), dtype=complex)
SIG = [np.array([[0, 1], [1, 0]], dtype=complex), np.array([[0, -1j], [1j, 0]], dtype=complex),
       np.array([[1, 0], [0, -1]], dtype=complex)]
G = [np.block([[I2, Z2], [Z2, -I2]])] + [np.block([[Z2, s], [-s, Z2]]) for s in SIG]   # Dirac rep
G5 = 1j * G[0] @ G[1] @ G[2] @ G[3]
PL = 0.5 * (np.eye(4) - G5)
PR = 0.5 * (np.eye(4) + G5)
METRIC = np.diag([1.0, -1.0, -1.0, -1.0])


def slash(p):
    return G[0] * p[0] - G[1] * p[1] - G[2] * p[2] - G[3] * p[3]


def mdot(a, b):
    return a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3]


def lorentz_contract(A, B):
    """sum_{mu,nu} A[mu][nu] B_{mu nu} for rank-2 tensors given with upper indices."""
    tot = 0.0
    for mu in range(4):
        for nu in range(4):
            tot += A[mu][nu] * B[mu][nu] * METRIC[mu, mu] * METRIC[nu, nu]
    return tot


def massless(E, cth, phi):
    sth = np.sqrt(max(0.0, 1.0 - cth * cth))
    return np.array([E, E * sth * np.cos(phi), E * sth * np.sin(phi), E * cth])


def random_massless(rng, scale=100.0):
    return massless(scale * (0.2 + rng.random()), 2 * rng.random() - 1, 2 * np.pi * rng.random())


def boost(p, b):
    """boost four-vector p by velocity vector b."""
    b = np.asarray(b, dtype=float)
    b2 = b @ b
    if b2 == 0:
        return np.array(p, dtype=float)
    g = 1.0 / np.sqrt(1.0 - b2)
    bp = b @ p[1:]
    out = np.empty(4)
    out[0] = g * (p[0] + bp)
    out[1:] = p[1:] + ((g - 1.0) * bp / b2 + g * p[0]) * b
    return out


def two_body_decay(P, m1, m2, cth, phi):
    """decay of four-momentum P into masses m1, m2 with rest-frame angles (cth, phi)."""
    M = np.sqrt(mdot(P, P))
    k = np.sqrt(max(0.0, (M * M - (m1 + m2) ** 2) * (M * M - (m1 - m2) ** 2))) / (2 * M)
    sth = np.sqrt(max(0.0, 1 - cth * cth))
    n = np.array([sth * np.cos(phi), sth * np.sin(phi), cth])
    p1 = np.concatenate([[np.sqrt(k * k + m1 * m1)], k * n])
    p2 = np.concatenate([[np.sqrt(k * k + m2 * m2)], -k * n])
    b = P[1:] / P[0]
    return boost(p1, b), boost(p2, b)
