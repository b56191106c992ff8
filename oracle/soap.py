"""float64 oracle of the SOAP optimizer step, Eqs. (12)-(13).  TEST INFRASTRUCTURE, NOT PRODUCT CODE (same
rules as the rest of ``oracle/``).  Plain numpy, one statement per line of the paper's equations, in the paper's order and
notation; the matrix products and the symmetric eigensolver are library routines (numpy / LAPACK), as the tier allows.

Readings:
  S21  M in "M' <- Q_L^T M Q_R" is the first moment of Eq. (10), kept in the original basis: M <- b1 M + (1 - b1) G, then
       rotated; V' lives in the rotated basis; the hats are Eq. (10)'s bias corrections with the step number i >= 1.
  S22  eps is inside the square root, N' = Mhat'/sqrt(Vhat' + eps), as Eq. (13) prints it (Eq. (11) has it outside; G4).
  S23  Q_L, Q_R are the full sets of orthonormal eigenvectors (columns) of the symmetric matrices L, R.  Their signs are
       free and do not change the update N (G', M', N' change sign together, V' holds squares); their order is the
       eigensolver's (ascending eigenvalues) and matters to V', so a caller keeps one convention.

Pins (tests/test_oracle_soap.py): with identity bases the step is Adam with eps inside the root, checked against its closed
form; a rank-one gradient a b^T gives the normalised rank-one update a_hat b_hat^T on the first step (closed form; Adam
would give sign(a_i b_j)); the whole recursion is equivariant under G -> U G W for orthogonal U, W (every transpose and
side of a product in Eqs. (12)-(13) matters to that); L, R stay symmetric positive semi-definite with trace L = trace R.
"""
from __future__ import annotations

import numpy as np


def soap_accumulate(L, R, G, b2: float = 0.999):
    """Eq. (12): L <- b2 L + (1 - b2) G G^T,  R <- b2 R + (1 - b2) G^T G."""
    L, R, G = (np.asarray(a, dtype=np.float64) for a in (L, R, G))
    L = b2 * L + (1.0 - b2) * (G @ G.T)
    R = b2 * R + (1.0 - b2) * (G.T @ G)
    return L, R


def soap_eigenbasis(A):
    """Eigenvectors of a symmetric accumulator: columns of Q, ascending eigenvalues w (LAPACK, S23)."""
    w, Q = np.linalg.eigh(np.asarray(A, dtype=np.float64))
    return Q, w


def soap_step(C, M, Vp, G, QL, QR, i: int, b1: float = 0.9, b2: float = 0.999, lr: float = 1e-3, eps: float = 1e-8):
    """Eq. (13) at step i >= 1 with the given bases; returns the new (C, M, V')."""
    C, M, Vp, G, QL, QR = (np.asarray(a, dtype=np.float64) for a in (C, M, Vp, G, QL, QR))
    M = b1 * M + (1.0 - b1) * G                       # Eq. (10), original basis (S21)
    Gp = QL.T @ G @ QR                                # G' <- Q_L^T G Q_R
    Mp = QL.T @ M @ QR                                # M' <- Q_L^T M Q_R
    Vp = b2 * Vp + (1.0 - b2) * Gp ** 2               # V' <- b2 V' + (1 - b2) (G')^2
    Mh = Mp / (1.0 - b1 ** i)                         # hats: Eq. (10)
    Vh = Vp / (1.0 - b2 ** i)
    Np = Mh / np.sqrt(Vh + eps)                       # N' <- Mhat'/sqrt(Vhat' + eps)   (S22)
    N = QL @ Np @ QR.T                                # N <- Q_L N' Q_R^T
    C = C - lr * N                                    # C <- C - eta N
    return C, M, Vp
