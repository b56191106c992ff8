"""The pieces composed into the paper's design loop on the GPU -- beta from Eq. (14), eps_hat and dF/dC from
given fields (Eq. (1)), the unbinarity feeding Eq. (15), an Adam or a SOAP step on C -- against the same loop written with
the float64 oracle.  There is no solver here: the fields are fixed synthetic arrays, so the objective is the linear
functional F(C) = sum_pairs -2 Re <E_F (.) E_A, eps_hat(C, beta)>, whose gradient Eq. (1) is; both sides minimise it."""
import numpy as np
import pytest
import torch

import oracle as O
from gpu_common import dev, oracle_cfg, rand_C, rand_fields
from paper_2505_03352_b200 import binding as B

pytestmark = pytest.mark.gpu

KW = dict(mx=20, my=18, nz=8, z_lo=2.25, z_hi=5.75, filter_radius=3.0, normal_delta=1e-8)
N_ITER, BETA_MIN, BETA_MAX0, GAMMA, U0, LR = 8, 4.0, 40.0, 0.9, 0.05, 0.02


def objective(eps, EF, EA):
    return sum(float(np.sum(-2.0 * np.real(f.astype(np.complex128) * a.astype(np.complex128)) * eps)) for f, a in zip(EF, EA))


@pytest.mark.parametrize("optimizer", ["adam", "soap"])
def test_design_loop_follows_the_oracle_loop(optimizer):
    cfg = B.make_config(**KW)
    oc = oracle_cfg(cfg)
    C0 = rand_C(cfg, 81)[0]
    EF, EA = rand_fields(cfg, 2, 82)
    dEF, dEA = [dev(f) for f in EF], [dev(f) for f in EA]
    f0, a0 = [f[0] for f in EF], [a[0] for a in EA]
    plan = B.Plan(cfg)
    # GPU state
    C = dev(C0[None].copy())
    M, V = torch.zeros_like(C), torch.zeros_like(C)
    soap = B.Soap(cfg.mx, cfg.my)
    t, bmax = 1.0, BETA_MAX0
    # oracle state
    Co, Mo, Vo = C0.astype(np.float64), np.zeros(C0.shape), np.zeros(C0.shape)
    Lo, Ro = np.zeros((cfg.mx, cfg.mx)), np.zeros((cfg.my, cfg.my))
    to, bmaxo = 1.0, BETA_MAX0
    F = []
    for i in range(1, N_ITER + 1):
        beta = B.beta_schedule(BETA_MIN, bmax, i, N_ITER)
        beta_o = O.beta_schedule(BETA_MIN, bmaxo, i, N_ITER)
        assert abs(beta - beta_o) < 1e-4 * beta_o
        eps, g = plan.eps_forward_vjp(C, beta, dEF, dEA)
        u = float(plan.unbinarity(C, beta)[0])
        go = O.vjp(oc, Co.astype(np.float32), beta_o, f0, a0)
        uo = O.unbinarity(oc, Co.astype(np.float32), beta_o)
        F.append(objective(eps[0].cpu().numpy().astype(np.float64), f0, a0))
        t, bmax = B.beta_update(t, bmax, GAMMA, u, U0, beta)
        to, bmaxo = O.beta_update(to, bmaxo, GAMMA, uo, U0, beta_o)
        if optimizer == "adam":
            B.adam_step(C, M, V, g, i, lr=LR)
            Co, Mo, Vo = O.adam_step(Co, Mo, Vo, go, i, lr=LR)
        else:
            # eps well above the square of float32 noise on G' (~1e-7 |G|): the rotated gradient is nearly diagonal in the first
            # iterations and Eq. (13) divides its noise entries by sqrt(noise^2 + eps)
            if i == 1:
                eps_soap = 1e-2 * float(np.mean(go ** 2))
            soap.accumulate(g[0], 0.95)
            soap.refresh()
            soap.update(C[0], g[0], b2=0.95, lr=LR, eps=eps_soap)
            Lo, Ro = O.soap_accumulate(Lo, Ro, go, 0.95)
            Co, Mo, Vo = O.soap_step(Co, Mo, Vo, go, O.soap_eigenbasis(Lo)[0], O.soap_eigenbasis(Ro)[0], i, 0.9, 0.95, LR, eps_soap)
        # the control variables stay together: steps are ~ LR = 2e-2 per iteration.  SOAP's rotated update N' = M'/sqrt(V' + eps) has
        # slope 1/sqrt(eps) at the entries that are zero in exact arithmetic, so the 1e-6 parity error of dF/dC shows more there
        err = np.max(np.abs(C[0].cpu().numpy().astype(np.float64) - Co))
        assert err < (2e-6 if optimizer == "adam" else 2e-5 * i), (optimizer, i, err)    # measured: 2.7e-7 / 9e-6 after 8 iterations
    assert abs(bmax - bmaxo) < 1e-3 * bmaxo and abs(t - to) < 1e-3 * to
    # both minimise F: for a fixed beta the first-order change is -LR * sum|g|-like, so F falls from the first iteration to the second
    assert F[1] < F[0]
