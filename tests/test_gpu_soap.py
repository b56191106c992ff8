"""GPU parity of the SOAP step (NEXT-3; Eqs. (12)-(13)) against the float64 oracle.  The eigenvectors are not
unique (signs; any basis inside a degenerate eigenspace), so the eigensolver is checked by what is unique -- the eigenvalues
and the defining properties of Q -- and the step by feeding both sides the same bases; whole iterations (each side with its
own eigensolver) are compared on the update, which does not depend on the signs (S23)."""
import numpy as np
import pytest
import torch

import oracle as O
from helpers import rel_inf
from paper_2505_03352_b200 import binding as B

pytestmark = pytest.mark.gpu


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


def host(t):
    return t.cpu().numpy().astype(np.float64)


@pytest.mark.parametrize("mx,my", [(5, 7), (64, 64), (70, 33), (250, 250), (129, 300)])
def test_accumulate_matches_oracle(mx, my):
    rng = np.random.default_rng(mx * 1000 + my)
    s = B.Soap(mx, my)
    L, R = np.zeros((mx, mx)), np.zeros((my, my))
    for _ in range(3):
        G = rng.standard_normal((mx, my)).astype(np.float32)
        s.accumulate(dev(G), 0.95)
        L, R = O.soap_accumulate(L, R, G, 0.95)
    assert rel_inf(host(s.L), L) < 2e-6 and rel_inf(host(s.R), R) < 2e-6
    assert torch.equal(s.L, s.L.T) and torch.equal(s.R, s.R.T)            # bitwise symmetric: the eigensolver reads one triangle


@pytest.mark.parametrize("n", [1, 6, 64, 250])
def test_eigensolver_by_its_defining_properties(n):
    rng = np.random.default_rng(n)
    X = rng.standard_normal((n, n + 3))
    A = (X @ X.T / (n + 3)).astype(np.float32)
    A = ((A + A.T) / 2).astype(np.float32)
    s = B.Soap(n, n)
    Q, w = torch.empty(n, n, device="cuda"), torch.empty(n, device="cuda")
    dA = dev(A)
    s.eigh(dA, Q, w, check=True)             # the solver status word (epsgrad_soap_eigh_info) must say "converged"
    torch.cuda.synchronize()
    assert torch.equal(dA, dev(A))                                          # the input is not written
    Qh, wh = host(Q), host(w)
    w_ref = np.linalg.eigvalsh(A.astype(np.float64))
    scale = np.abs(w_ref).max()
    assert np.all(np.diff(wh) >= 0) and np.max(np.abs(wh - w_ref)) < 1e-5 * scale
    assert np.max(np.abs(Qh.T @ Qh - np.eye(n))) < 1e-5                      # orthonormal columns
    assert np.max(np.abs(A.astype(np.float64) @ Qh - Qh * wh)) < 2e-5 * scale   # A q_j = w_j q_j, column by column


@pytest.mark.parametrize("mx,my", [(5, 7), (70, 33), (250, 250)])
def test_step_matches_oracle_given_the_same_bases(mx, my):
    rng = np.random.default_rng(7 + mx)
    orth = lambda n: np.linalg.qr(rng.standard_normal((n, n)))[0].astype(np.float32)
    C = rng.random((mx, my)).astype(np.float32)
    M0 = (0.1 * rng.standard_normal((mx, my))).astype(np.float32)
    V0 = (rng.random((mx, my)) * 0.5).astype(np.float32)
    G = rng.standard_normal((mx, my)).astype(np.float32)
    QL, QR = orth(mx), orth(my)
    s = B.Soap(mx, my)
    s.M.copy_(dev(M0)); s.Vp.copy_(dev(V0)); s.QL.copy_(dev(QL)); s.QR.copy_(dev(QR))
    s.step = 4
    dC = dev(C)
    s.update(dC, dev(G), b1=0.9, b2=0.99, lr=0.01, eps=1e-8)
    C1, M1, V1 = O.soap_step(C, M0, V0, G, QL, QR, 5, 0.9, 0.99, 0.01, 1e-8)
    assert rel_inf(host(s.M), M1) < 1e-6 and rel_inf(host(s.Vp), V1) < 1e-5
    # compare the update, not C (C - lr N would hide N behind C's magnitude)
    N, N_ref = (C.astype(np.float64) - host(dC)) / 0.01, (C - C1) / 0.01
    assert rel_inf(N, N_ref) < 1e-4, rel_inf(N, N_ref)


def test_iterations_match_oracle_each_side_with_its_own_eigensolver():
    # Four full iterations (accumulate, eigenvectors, step).  In the exact eigenbases of G G^T and G^T G the rotated gradient
    # of the first step is diagonal (they are the singular vectors of G), and Eq. (13) turns every other entry -- exactly 0,
    # rounding noise in practice -- into noise/sqrt(noise^2 + eps): ~1e-13 in float64 but 1e-7/sqrt(eps) in float32.  The
    # comparison therefore uses an eps well above float32 noise squared; with App. B's 1e-8 the first SOAP update is
    # ill-conditioned on any float32 implementation.
    rng = np.random.default_rng(21)
    mx, my = 24, 17
    base = rng.standard_normal((mx, my))
    s = B.Soap(mx, my)
    dC = torch.zeros(mx, my, device="cuda")
    C, M, Vp, L, R = np.zeros((mx, my)), np.zeros((mx, my)), np.zeros((mx, my)), np.zeros((mx, mx)), np.zeros((my, my))
    for i in range(1, 5):
        G = (base + 0.3 * rng.standard_normal((mx, my))).astype(np.float32)
        s.accumulate(dev(G), 0.9)
        s.refresh()
        s.update(dC, dev(G), b1=0.9, b2=0.9, lr=0.05, eps=1e-2)
        L, R = O.soap_accumulate(L, R, G, 0.9)
        QL, QR = O.soap_eigenbasis(L)[0], O.soap_eigenbasis(R)[0]
        C, M, Vp = O.soap_step(C, M, Vp, G, QL, QR, i, 0.9, 0.9, 0.05, 1e-2)
        err = rel_inf(host(dC), C)
        assert err < 5e-4, (i, err)                    # float32 eigenvectors: error ~ 1e-7 / relative spectral gap
    assert rel_inf(host(s.M), M) < 1e-6


def test_argument_checks():
    s = B.Soap(4, 4)
    L = B.lib()
    z = torch.zeros(4, 4, device="cuda")
    assert L.epsgrad_soap_accumulate(None, z.data_ptr(), z.data_ptr(), 4, 4, 0.9, None) == B.EINVAL
    assert L.epsgrad_soap_accumulate(z.data_ptr(), z.data_ptr(), z.data_ptr(), 4, 4, 1.0, None) == B.EINVAL
    assert L.epsgrad_soap_step(z.data_ptr(), z.data_ptr(), z.data_ptr(), z.data_ptr(), z.data_ptr(), z.data_ptr(), 4, 4, 0,
                               0.9, 0.99, 0.01, 1e-8, s._work.data_ptr(), s._work.numel(), None) == B.EINVAL
    assert L.epsgrad_soap_step(z.data_ptr(), z.data_ptr(), z.data_ptr(), z.data_ptr(), z.data_ptr(), z.data_ptr(), 4, 4, 1,
                               0.9, 0.99, 0.01, 1e-8, s._work.data_ptr(), 16, None) == B.ENOWORKSPACE
    assert L.epsgrad_soap_eigh(z.data_ptr(), z.data_ptr(), z.data_ptr(), 4, None, 0, None) == B.ENOWORKSPACE
    assert L.epsgrad_soap_step_workspace_bytes(0, 4) == 0
