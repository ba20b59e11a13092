"""GPU parity of full time steps forward + backward (BASELINE.json configs[1] shape): the loss, the end-to-end
parameter gradient dJ/dtheta (north_star: within 1e-3) and dJ/dU0, C ABI path vs the fp64 oracle's rollout on the
same seeded geometry."""
import numpy as np
import pytest

from oracle import nf_oracle as orc
from paper_2405_14903_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available()
    return t


@pytest.fixture(scope="module")
def api():
    from paper_2405_14903_b200 import api as a
    a.load_library()
    return a


@pytest.mark.parametrize("n,nsteps,u0_amp", [(32, 4, 0.0), (24, 3, 0.2)])
def test_rollout_loss_and_gradients_match_oracle(torch, api, n, nsteps, u0_amp):
    from paper_2405_14903_b200 import rollout as ro
    P = wl.config2_params(n)
    bc = orc.BC(P["bc_types"], P["bc_values"])
    rng = np.random.default_rng(1002)
    U0 = [(u0_amp * rng.standard_normal(s)).astype(np.float32) for s in wl.face_shapes(n, n, n)]
    theta = P["theta"]
    geom = {s: wl.config2_solid(P, s, theta) for s in range(1, nsteps + 1)}  # fp32 phi / u_s: the SAME arrays on both sides
    lo, hi = P["loss_lo"], P["loss_hi"]

    # oracle
    Jo, dJo, gU0o = orc.rollout(U0, lambda s: geom[s], nsteps, P["dt"], P["dx"], P["dt_over_rho"], bc,
                                orc.loss_sum_u2(lo, hi))

    # CUDA path
    d = lambda a: None if a is None else torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()
    g = api.Grid(n, n, n, P["dx"])
    g.set_dt_rho(P["dt_over_rho"])
    dgeom = {s: (d(v[0]), [d(a) for a in v[1]], d(v[2]), [d(a) for a in v[3]]) for s, v in geom.items()}

    def loss(U):
        blk = U[0][lo:hi, lo:hi, lo:hi].double()
        G = [torch.zeros_like(a) for a in U]
        G[0][lo:hi, lo:hi, lo:hi] = (2.0 * blk).float()
        return (blk * blk).sum(), G

    Jg, dJg, gU0g = ro.rollout(g, [d(a) for a in U0], lambda s: dgeom[s], nsteps, P["dt"], loss, tol=1e-6, maxit=200)
    g.close()
    assert Jo > 0
    assert abs(Jg - Jo) <= 1e-4 * abs(Jo), (Jg, Jo)
    assert abs(dJg - dJo) <= 1e-3 * abs(dJo), (dJg, dJo)
    num = np.sqrt(sum(np.sum((a.cpu().numpy().astype(np.float64) - b) ** 2) for a, b in zip(gU0g, gU0o)))
    den = np.sqrt(sum(np.sum(b ** 2) for b in gU0o))
    # With the fluid at rest every back-traced point sits exactly ON a lattice node, where trilinear interpolation
    # has a kink: the one-sided position derivative taken there depends on rounding, so dJ/dU0 is only compared for
    # the generic initial velocity.
    if u0_amp > 0 and den > 0:
        assert num <= 1e-3 * den, num / den
