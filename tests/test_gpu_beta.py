"""GPU parity of the beta-related outputs (NEXT-2): d F/d beta and the unbinarity u(beta) against the float64
oracle, with and without the morphological filters; the host-side beta schedule against the oracle's Eqs. (14)-(15)."""
import numpy as np
import pytest
import torch

import oracle as O
from gpu_common import TOL_GRAD, dev, oracle_cfg, rand_C, rand_fields
from helpers import rel_inf
from paper_2505_03352_b200 import binding as B

pytestmark = pytest.mark.gpu

CASES = [
    dict(mx=9, my=7, nz=8, z_lo=2.25, z_hi=5.75, filter_radius=3.0),
    dict(batch=2, mx=37, my=29, nz=16, z_lo=6.25, z_hi=9.75, filter_radius=4.0),
    dict(batch=2, mx=33, my=21, nz=16, z_lo=6.25, z_hi=9.75, filter_radius=4.0, morph_diameter=4.0),
    dict(mx=20, my=18, nz=8, z_lo=2.25, z_hi=5.75, subpixel=4, filter_radius=3.0, morph_diameter=2.5),
    dict(mx=250, my=250, nz=64, z_lo=28.25, z_hi=35.75, filter_radius=8.0),
]


@pytest.mark.parametrize("kw", CASES)
@pytest.mark.parametrize("beta", [6.0, 20.0])
def test_dbeta_and_unbinarity_match_oracle(kw, beta):
    cfg = B.make_config(**kw)
    C = rand_C(cfg, 41)
    EF, EA = rand_fields(cfg, 2, 42)
    plan = B.Plan(cfg)
    dEF, dEA = [dev(f) for f in EF], [dev(f) for f in EA]
    g, db = plan.eps_vjp_beta(dev(C), beta, dEF, dEA)
    u = plan.unbinarity(dev(C), beta)
    g0 = plan.eps_vjp(dev(C), beta, dEF, dEA)
    g2, db2 = plan.eps_vjp_beta(dev(C), beta, dEF, dEA)
    torch.cuda.synchronize()
    assert torch.equal(g, g0) and torch.equal(g, g2) and torch.equal(db, db2)          # same gradient; reproducible sums
    oc = oracle_cfg(cfg)
    for b in range(cfg.batch):
        g_ref, db_ref = O.vjp_beta(oc, C[b], beta, [f[b] for f in EF], [f[b] for f in EA])
        u_ref = O.unbinarity(oc, C[b], beta)
        assert rel_inf(g[b].cpu().numpy().astype(np.float64), g_ref) < TOL_GRAD
        # d F/d beta is a sum of signed per-pixel terms: compare against the sum of their magnitudes' scale, max |dF/dC| * N
        scale = max(abs(db_ref), 1e-3 * np.abs(g_ref).sum())
        assert abs(float(db[b]) - db_ref) < TOL_GRAD * scale, (float(db[b]), db_ref)
        assert abs(float(u[b]) - u_ref) < 1e-5 * max(u_ref, 1e-3), (float(u[b]), u_ref)


def test_beta_schedule_matches_oracle():
    for i in range(0, 101, 7):
        assert abs(B.beta_schedule(10.0, 150.0, i, 100) - O.beta_schedule(10.0, 150.0, i, 100)) < 1e-12
    t, bm = 1.0, 60.0
    to, bo = t, bm
    for it in range(50):
        beta, u = 10.0 + it, 1.0 / (1.0 + 0.3 * (10.0 + it))
        t, bm = B.beta_update(t, bm, 0.95, u, 0.01, beta)
        to, bo = O.beta_update(to, bo, 0.95, u, 0.01, beta)
        assert abs(t - to) < 1e-13 and abs(bm - bo) < 1e-10
    with pytest.raises(B.EpsgradError):
        B.beta_update(1.0, 50.0, 0.95, 0.0, 0.01, 10.0)


def test_adam_steps_match_oracle():
    rng = np.random.default_rng(51)
    shape = (2, 37, 29)
    C0 = rng.random(shape).astype(np.float32)
    C, M, V = dev(C0.copy()), torch.zeros(shape, device="cuda"), torch.zeros(shape, device="cuda")
    Co, Mo, Vo = C0.astype(np.float64), np.zeros(shape), np.zeros(shape)
    for i in range(1, 21):
        G = (rng.standard_normal(shape) * (0.01 + 0.1 * i)).astype(np.float32)
        B.adam_step(C, M, V, dev(G), i)
        Co, Mo, Vo = O.adam_step(Co, Mo, Vo, G, i)
        assert np.max(np.abs(C.cpu().numpy() - Co)) < 2e-6
        assert rel_inf(M.cpu().numpy().astype(np.float64), Mo) < 1e-5 and rel_inf(V.cpu().numpy().astype(np.float64), Vo) < 1e-5
    with pytest.raises(B.EpsgradError):
        B.adam_step(C, M, V, C, 0)
