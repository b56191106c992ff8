"""Pins of the oracle's SOAP step (NEXT-3; Eqs. (12)-(13); readings S21-S23) against things other than itself:
closed forms, the Adam special case, and the equivariance under rotations that distinguishes SOAP from Adam."""
import numpy as np

import oracle as O


def _orth(n, rng):
    q, r = np.linalg.qr(rng.standard_normal((n, n)))
    return q * np.sign(np.diag(r))


def test_identity_bases_give_adam_with_eps_inside_the_root():
    rng = np.random.default_rng(1)
    mx, my = 5, 7
    C, M, V = rng.random((mx, my)), 0.1 * rng.standard_normal((mx, my)), rng.random((mx, my))
    G = rng.standard_normal((mx, my))
    b1, b2, lr, eps, i = 0.9, 0.99, 0.01, 1e-6, 4
    C1, M1, V1 = O.soap_step(C, M, V, G, np.eye(mx), np.eye(my), i, b1, b2, lr, eps)
    # Eq. (10) written out element by element, eps inside the root (S22)
    for a in range(mx):
        for b in range(my):
            m = b1 * M[a, b] + (1 - b1) * G[a, b]
            v = b2 * V[a, b] + (1 - b2) * G[a, b] ** 2
            c = C[a, b] - lr * (m / (1 - b1 ** i)) / np.sqrt(v / (1 - b2 ** i) + eps)
            assert abs(M1[a, b] - m) < 1e-15 and abs(V1[a, b] - v) < 1e-15 and abs(C1[a, b] - c) < 1e-15
    # and, for eps -> 0, the library's Adam (eps outside the root, Eq. (11)) agrees
    C2, M2, V2 = O.adam_step(C, M, V, G, i, b1, b2, lr, 0.0)
    C3, _, _ = O.soap_step(C, M, V, G, np.eye(mx), np.eye(my), i, b1, b2, lr, 0.0)
    assert np.max(np.abs(C2 - C3)) < 1e-14 and np.max(np.abs(M2 - M1)) < 1e-15 and np.max(np.abs(V2 - V1)) < 1e-15


def test_rank_one_gradient_gives_the_normalised_rank_one_update():
    # G = a b^T: L = (1-b2)|b|^2 a a^T, R = (1-b2)|a|^2 b b^T; in their eigenbases G' has the single entry |a||b|, so on the first
    # step N' = 1 there (0 elsewhere: 0/sqrt(0 + eps)) and N = a_hat b_hat^T, whatever the scale of G.  Adam gives sign(a_i b_j).
    rng = np.random.default_rng(2)
    a, b = rng.standard_normal(6), rng.standard_normal(4)
    G = 37.0 * np.outer(a, b)
    L, R = O.soap_accumulate(np.zeros((6, 6)), np.zeros((4, 4)), G, 0.999)
    assert np.allclose(L, 0.001 * 37.0 ** 2 * (b @ b) * np.outer(a, a), rtol=1e-12, atol=0)
    assert np.allclose(R, 0.001 * 37.0 ** 2 * (a @ a) * np.outer(b, b), rtol=1e-12, atol=0)
    QL, wl = O.soap_eigenbasis(L)
    QR, wr = O.soap_eigenbasis(R)
    assert abs(wl[-1] - np.trace(L)) < 1e-9 * wl[-1] and abs(wr[-1] - np.trace(R)) < 1e-9 * wr[-1]
    C0 = rng.random((6, 4))
    C1, M1, V1 = O.soap_step(C0, np.zeros((6, 4)), np.zeros((6, 4)), G, QL, QR, 1, 0.9, 0.999, 0.05, 1e-12)
    N = (C0 - C1) / 0.05
    ref = np.outer(a / np.linalg.norm(a), b / np.linalg.norm(b))
    assert np.max(np.abs(N - ref)) < 1e-7
    assert np.max(np.abs(M1 - 0.1 * G)) < 1e-13 * np.abs(G).max()


def _run(Gs, C0, b1, b2, lr, eps):
    mx, my = C0.shape
    C, M, Vp = C0.copy(), np.zeros((mx, my)), np.zeros((mx, my))
    L, R = np.zeros((mx, mx)), np.zeros((my, my))
    for i, G in enumerate(Gs, start=1):
        L, R = O.soap_accumulate(L, R, G, b2)
        QL, _ = O.soap_eigenbasis(L)
        QR, _ = O.soap_eigenbasis(R)
        C, M, Vp = O.soap_step(C, M, Vp, G, QL, QR, i, b1, b2, lr, eps)
    return C, M, L, R


def test_recursion_is_equivariant_under_rotations_of_the_gradient():
    # Rotate every gradient, G -> U G W^T with orthogonal U, W: then L -> U L U^T, R -> W R W^T, Q_L -> U Q_L, Q_R -> W Q_R, the
    # rotated-basis quantities G', M', V', N' do not change at all, and the update rotates with the gradient: C - C0 -> U (C - C0) W^T.
    # A transposed factor, a swapped side or Q_L used for Q_R anywhere in Eqs. (12)-(13) breaks this; Adam is not equivariant.
    rng = np.random.default_rng(3)
    mx, my = 5, 4
    Gs = [rng.standard_normal((mx, my)) for _ in range(4)]
    U, W = _orth(mx, rng), _orth(my, rng)
    C0 = np.zeros((mx, my))
    C, M, L, R = _run(Gs, C0, 0.9, 0.95, 0.02, 1e-10)
    Cr, Mr, Lr, Rr = _run([U @ G @ W.T for G in Gs], C0, 0.9, 0.95, 0.02, 1e-10)
    assert np.max(np.abs(Cr - U @ C @ W.T)) < 1e-9 * np.abs(C).max()
    assert np.max(np.abs(Mr - U @ M @ W.T)) < 1e-12 and np.max(np.abs(Lr - U @ L @ U.T)) < 1e-12
    assert np.max(np.abs(Rr - W @ R @ W.T)) < 1e-12
    # the Adam step is not: the same rotation changes its update
    Ca = np.zeros((mx, my)); Ma = np.zeros((mx, my)); Va = np.zeros((mx, my))
    Cb = np.zeros((mx, my)); Mb = np.zeros((mx, my)); Vb = np.zeros((mx, my))
    for i, G in enumerate(Gs, start=1):
        Ca, Ma, Va = O.adam_step(Ca, Ma, Va, G, i, 0.9, 0.95, 0.02, 1e-10)
        Cb, Mb, Vb = O.adam_step(Cb, Mb, Vb, U @ G @ W.T, i, 0.9, 0.95, 0.02, 1e-10)
    assert np.max(np.abs(Cb - U @ Ca @ W.T)) > 1e-3


def test_accumulators_stay_symmetric_psd_with_equal_traces():
    rng = np.random.default_rng(4)
    L, R = np.zeros((6, 6)), np.zeros((3, 3))
    for _ in range(5):
        L, R = O.soap_accumulate(L, R, rng.standard_normal((6, 3)), 0.9)
    assert np.array_equal(L, L.T) or np.max(np.abs(L - L.T)) < 1e-15
    assert abs(np.trace(L) - np.trace(R)) < 1e-12 * np.trace(L)                     # both are the averaged |G|_F^2
    QL, wl = O.soap_eigenbasis(L)
    assert wl.min() > -1e-12 and np.max(np.abs(QL.T @ QL - np.eye(6))) < 1e-12
    assert np.max(np.abs(QL @ np.diag(wl) @ QL.T - L)) < 1e-12 * wl.max()
    assert np.all(np.diff(wl) >= 0)


def test_eigenvector_signs_do_not_change_the_update():
    rng = np.random.default_rng(5)
    mx, my = 4, 6
    G, M, Vp, C = (rng.standard_normal((mx, my)) for _ in range(4))
    Vp = Vp ** 2
    QL, QR = _orth(mx, rng), _orth(my, rng)
    sL, sR = np.array([1, -1, -1, 1.0]), np.array([-1, 1, 1, -1, 1, -1.0])
    a = O.soap_step(C, M, Vp, G, QL, QR, 3)
    b = O.soap_step(C, M, Vp, G, QL * sL, QR * sR, 3)
    for x, y in zip(a, b):
        assert np.max(np.abs(x - y)) < 1e-13
