"""GPU parity of the parametric geometry (include/nf.h nf_geom_*) against
oracle/nf_geom_oracle.py on the same seeded fp32 parameter vectors, through the C ABI.

Tolerances: coordinates are O(1); the device rounds the vertices (built in fp64) and the node
coordinates to fp32 and scans in fp32, so phi carries a few ulp of 1: atol 2e-6.  The unit normal (x - q)/|x - q| and
with it U_s and the gradients lose relative accuracy like eps / |d| next to the surface: velocities are compared at
1e-4 relative to max|U_s| where |d| > 1e-3 and at 2e-2 elsewhere.  Where two edges are equidistant (the medial axis)
the closest edge, hence the normal, is not unique and fp32 may break the tie the other way: up to 0.1 % of the faces
may disagree, at least 4 on a small grid (phi itself is continuous there and is compared everywhere)."""
import numpy as np
import pytest

from oracle import nf_geom_oracle as G
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


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


CASES = {
    # name: (nx, ny, nz, dx, K, N, M, z0, z1, centre, radius)
    "ragged_k3": (40, 36, 28, 1.0 / 40, 3, 5, 12, 0.13, 0.61, (0.5, 0.45), 0.27),
    "wide_k1": (72, 40, 12, 1.0 / 72, 1, 4, 8, 0.04, 0.12, (0.5, 0.28), 0.2),
    "many_edges": (20, 24, 8, 1.0 / 24, 2, 32, 64, 0.1, 0.3, (0.42, 0.5), 0.3),   # N M = 2048: opt-in shared memory
    "plane_2d": (48, 48, 1, 1.0 / 48, 1, 6, 16, -1.0, 2.0, (0.5, 0.5), 0.3),
}


def make(api, name):
    nx, ny, nz, dx, K, N, M, z0, z1, c, r = CASES[name]
    dx = float(np.float32(dx))
    p = wl.geom_random_params(2000 + len(name), K, N, z0, z1, c, r)
    return api.Grid(nx, ny, nz, dx), (nx, ny, nz, dx, K, N, M), p


@pytest.mark.parametrize("name", list(CASES))
@pytest.mark.parametrize("complement", [False, True])
def test_sdf_matches_oracle(torch, api, name, complement):
    g, (nx, ny, nz, dx, K, N, M), p = make(api, name)
    sdf = torch.full(g.shape_sdf, 9.0, dtype=torch.float32, device="cuda")
    g.geom_sdf(p, K, N, M, sdf, complement)
    ref = G.sdf_nodes(p.astype(np.float64), K, N, M, nx, ny, nz, dx, complement)
    got = sdf.cpu().numpy().astype(np.float64)
    assert np.max(np.abs(got - ref)) < 2e-6
    assert (ref < 0).any() and (ref > 0).any()
    g.close()


@pytest.mark.parametrize("name", ["ragged_k3", "wide_k1", "many_edges"])
@pytest.mark.parametrize("complement", [False, True])
def test_sdf_adjoint_matches_oracle(torch, api, name, complement):
    g, (nx, ny, nz, dx, K, N, M), p = make(api, name)
    rng = np.random.default_rng(77)
    gphi = rng.standard_normal((nz + 1, ny + 1, nx + 1)).astype(np.float32)
    # like dJ/dphi of the weight builder: only nodes next to the surface carry a gradient, plus a dense case below
    ref_phi = G.sdf_nodes(p.astype(np.float64), K, N, M, nx, ny, nz, dx, complement)
    for mask in (np.abs(ref_phi) < 2 * dx, np.ones_like(ref_phi, dtype=bool)):
        gp = np.where(mask, gphi, 0.0).astype(np.float32)
        got = g.geom_sdf_adjoint(p, K, N, M, dev(torch, gp), complement)
        ref = G.sdf_nodes_adjoint(p.astype(np.float64), K, N, M, nx, ny, nz, dx, gp.astype(np.float64), complement)
        assert np.max(np.abs(ref)) > 0
        assert np.max(np.abs(got - ref)) < 2e-4 * np.max(np.abs(ref))
    # nothing upstream -> exactly zero
    assert not g.geom_sdf_adjoint(p, K, N, M, torch.zeros(g.shape_sdf, device="cuda"), complement).any()
    g.close()


def test_csg_and_its_adjoint_are_exact(torch, api):
    g, (nx, ny, nz, dx, K, N, M), p = make(api, "ragged_k3")
    q = wl.geom_random_params(5, 1, 4, 0.3, 0.9, (0.62, 0.5), 0.2)
    a = torch.empty(g.shape_sdf, dtype=torch.float32, device="cuda")
    b = torch.empty_like(a)
    g.geom_sdf(p, K, N, M, a)
    g.geom_sdf(q, 1, 4, 10, b)
    an, bn = a.cpu().numpy(), b.cpu().numpy()
    gout = np.random.default_rng(3).standard_normal(an.shape).astype(np.float32)
    for op in ("union", "intersection"):
        out = torch.empty_like(a)
        g.geom_csg(op, a, b, out)
        assert np.array_equal(out.cpu().numpy(), G.csg(op, an, bn))
        ga, gb = torch.empty_like(a), torch.empty_like(a)
        g.geom_csg_adjoint(op, a, b, dev(torch, gout), ga, gb)
        ra, rb = G.csg_adjoint(op, an, bn, gout)
        assert np.array_equal(ga.cpu().numpy(), ra) and np.array_equal(gb.cpu().numpy(), rb)
    # in place
    c = a.clone()
    g.geom_csg("union", c, b, c)
    assert np.array_equal(c.cpu().numpy(), np.minimum(an, bn))
    g.close()


def face_distance(p, K, N, M, nx, ny, nz, dx, comp):
    """The primitive's signed distance at the face centres of family comp (from the oracle's public pieces)."""
    xi, xc = np.arange(nx + 1) * dx, (np.arange(nx) + 0.5) * dx
    yj, yc = np.arange(ny + 1) * dx, (np.arange(ny) + 0.5) * dx
    X, Y = np.meshgrid(*[(xi, yc), (xc, yj), (xc, yc)][comp], indexing="xy")
    zs = (np.arange(nz) + 0.5) * dx if comp < 2 else np.arange(nz + 1) * dx
    out = []
    for z in zs:
        c, r1, r2 = G.section_at(p, K, N, z)[:3]
        out.append(np.maximum(G.sdf2d(c, r1, r2, M, X, Y), max(p[0] - z, z - p[1])))
    return np.stack(out)


@pytest.mark.parametrize("name", ["ragged_k3", "wide_k1", "plane_2d"])
def test_velocity_matches_oracle(torch, api, name):
    g, (nx, ny, nz, dx, K, N, M), p = make(api, name)
    pd = wl.geom_random_rates(9, K, N, 0.2)
    p64, pd64 = p.astype(np.float64), pd.astype(np.float64)
    out = [torch.full(s, 5.0, dtype=torch.float32, device="cuda") for s in (g.shape_u, g.shape_v, g.shape_w)]
    g.geom_velocity(p, pd, K, N, M, *out)
    ref = G.solid_velocity_faces(p64, pd64, K, N, M, nx, ny, nz, dx)
    scale = max(np.max(np.abs(r)) for r in ref)
    assert scale > 0.05
    for comp in range(3):
        got = out[comp].cpu().numpy().astype(np.float64)
        d = face_distance(p64, K, N, M, nx, ny, nz, dx, comp)
        err = np.abs(got - ref[comp])
        bad = np.where(np.abs(d) > 1e-3, err > 1e-4 * scale, err > 2e-2 * scale)
        assert np.count_nonzero(bad) <= max(4, 1e-3 * bad.size), (comp, np.count_nonzero(bad), bad.size)
    # band: faces farther than the band keep their value; the others are as before
    band = 2.5 * dx
    keep = [torch.full(s, 7.0, dtype=torch.float32, device="cuda") for s in (g.shape_u, g.shape_v, g.shape_w)]
    g.geom_velocity(p, pd, K, N, M, *keep, band=band)
    for comp in range(3):
        d = face_distance(p64, K, N, M, nx, ny, nz, dx, comp)
        got = keep[comp].cpu().numpy()
        sure_out, sure_in = d > band + 1e-5, d < band - 1e-5
        assert np.all(got[sure_out] == 7.0)
        assert np.array_equal(got[sure_in], out[comp].cpu().numpy()[sure_in])
        assert sure_in.any() and sure_out.any()
    g.close()


@pytest.mark.parametrize("name", ["ragged_k3", "wide_k1"])
def test_velocity_adjoint_is_the_transpose(torch, api, name):
    g, (nx, ny, nz, dx, K, N, M), p = make(api, name)
    rng = np.random.default_rng(21)
    gs = [rng.standard_normal(s).astype(np.float32) for s in (g.shape_u, g.shape_v, g.shape_w)]
    band = 3.0 * dx
    got = g.geom_velocity_adjoint(p, K, N, M, *[dev(torch, a) for a in gs], band=band)
    # dot-product identity on the device path: <J pdot, g> = <pdot, J^T g>
    for seed in (1, 2):
        pd = wl.geom_random_rates(seed, K, N, 1.0)
        out = [torch.zeros(s, dtype=torch.float32, device="cuda") for s in (g.shape_u, g.shape_v, g.shape_w)]
        g.geom_velocity(p, pd, K, N, M, *out, band=band)
        lhs = sum(float((o.double() * dev(torch, a).double()).sum()) for o, a in zip(out, gs))
        rhs = float(got @ pd.astype(np.float64))
        assert abs(lhs - rhs) <= 1e-4 * max(abs(lhs), abs(rhs))
    # and against the oracle's transpose (faces within 1e-5 of the band edge may fall on either side: masked out)
    p64 = p.astype(np.float64)
    gm = []
    for comp in range(3):
        d = face_distance(p64, K, N, M, nx, ny, nz, dx, comp)
        gm.append(np.where(np.abs(d - band) < 1e-5, 0.0, gs[comp]).astype(np.float32))
    got = g.geom_velocity_adjoint(p, K, N, M, *[dev(torch, a) for a in gm], band=band)
    ref = G.solid_velocity_faces_adjoint(p64, K, N, M, nx, ny, nz, dx, *[a.astype(np.float64) for a in gm], band=band)
    assert np.max(np.abs(got - ref)) < 2e-3 * np.max(np.abs(ref))
    g.close()


def test_design_gradient_through_projection_matches_oracle(torch, api):
    """The co-design chain of PAPER.md:L132-141: params -> phi -> alpha -> projection -> J = 1/2 |U^{n+1}|^2 and back
    (nf_project_adjoint -> nf_weights_adjoint -> nf_geom_sdf_adjoint), device path vs the fp64 oracle chain; north_star's
    gradient tolerance 1e-3."""
    n, dx = 24, float(np.float32(1.0 / 24))
    K, N, M = 2, 5, 10
    p = wl.geom_random_params(31, K, N, 0.2, 0.8, (0.5, 0.5), 0.22)
    bc_t, bc_v = (1, 1, 0, 0, 0, 0), (1.0, 0.0, 0, 0, 0, 0)
    bc = orc.BC(bc_t, bc_v)
    rng = np.random.default_rng(5)
    U = [(0.3 * rng.standard_normal(s)).astype(np.float32) for s in wl.face_shapes(n, n, n)]
    # device
    g = api.Grid(n, n, n, dx)
    for f in range(6):
        g.set_domain_bc(f, bc_t[f], bc_v[f])
    sdf = torch.empty(g.shape_sdf, dtype=torch.float32, device="cuda")
    g.geom_sdf(p, K, N, M, sdf)
    g.set_solid(sdf, None, None, None)
    Ud = [dev(torch, a) for a in U]
    pr = torch.empty(g.shape_p, dtype=torch.float32, device="cuda")
    assert g.project(*Ud, pr, tol=1e-7, maxit=300) == 0
    J = 0.5 * sum(float((a.double() ** 2).sum()) for a in Ud)
    Gd = [a.clone() for a in Ud]
    ga = [torch.empty_like(a) for a in Ud]
    assert g.project_adjoint(*Gd, p_saved=pr, uhat=[dev(torch, a) for a in U], galpha=ga, gus=None, y_out=None,
                             tol=1e-7, maxit=300) == 0
    gsdf = torch.empty_like(sdf)
    g.weights_adjoint(*ga, gsdf)
    got = g.geom_sdf_adjoint(p, K, N, M, gsdf)
    # oracle; the weights are built from the device's fp32 phi (checked against the oracle's first) so that both sides
    # classify the same faces (alpha < 1e-4 -> 0 is a threshold: R4)
    p64 = p.astype(np.float64)
    phi = sdf.cpu().numpy().astype(np.float64)
    assert np.max(np.abs(phi - G.sdf_nodes(p64, K, N, M, n, n, n, dx))) < 2e-6
    alpha = orc.face_weights(phi, bc)
    Un, pref = orc.project(U, alpha, None, dx, 1.0, bc)
    Jref = 0.5 * sum(float((a ** 2).sum()) for a in Un)
    _, gA, _, _ = orc.project_adjoint(Un, alpha, pref, U, None, dx, 1.0, bc)
    gphi = orc.weights_adjoint(phi, *gA, bc)
    ref = G.sdf_nodes_adjoint(p64, K, N, M, n, n, n, dx, gphi)
    assert abs(J - Jref) < 1e-4 * Jref
    assert np.max(np.abs(ref)) > 0
    assert np.max(np.abs(got - ref)) < 1e-3 * np.max(np.abs(ref))
    g.close()


def test_geometry_error_codes(torch, api):
    g = api.Grid(8, 8, 8, 0.125)
    sdf = torch.empty(g.shape_sdf, dtype=torch.float32, device="cuda")
    p = wl.geom_random_params(1, 1, 4, 0.2, 0.8, (0.5, 0.5), 0.2)
    bad = p.copy(); bad[4] = -1.0
    with pytest.raises(api.NfError):
        g.geom_sdf(bad, 1, 4, 8, sdf)
    bad = p.copy(); bad[1] = bad[0]
    with pytest.raises(api.NfError):
        g.geom_sdf(bad, 1, 4, 8, sdf)
    with pytest.raises(api.NfError):
        g.geom_sdf(wl.geom_random_params(1, 1, 64, 0.2, 0.8, (0.5, 0.5), 0.2), 1, 64, 33, sdf)   # N M > 2048
    g.geom_sdf(p, 1, 4, 8, sdf)
    g.close()


def test_parametric_rollout_matches_oracle(torch, api):
    """Two full time steps with a static and a moving primitive: loss, dJ/dparams and dJ/dpdot of every primitive at
    every step, dJ/dU0 -- device path (paper_2405_14903_b200/rollout.py: C-ABI calls only) vs the oracle's
    rollout_parametric; north_star's tolerances (1e-4 loss and fields, 1e-3 gradients)."""
    from paper_2405_14903_b200 import rollout as ro
    n, dx = 24, float(np.float32(1.0 / 24))
    bc_t, bc_v = (1, 1, 0, 0, 0, 0), (1.0, 0.0, 0, 0, 0, 0)
    bc = orc.BC(bc_t, bc_v)
    rng = np.random.default_rng(8)
    U0 = [(0.2 * rng.standard_normal(s)).astype(np.float32) for s in wl.face_shapes(n, n, n)]
    pA = wl.geom_random_params(51, 2, 5, 0.21, 0.79, (0.36, 0.5), 0.17)
    pB = wl.geom_random_params(52, 1, 4, 0.3, 0.71, (0.7, 0.46), 0.12)
    dB = wl.geom_random_rates(53, 1, 4, 0.3)
    band, dt, nsteps = 3.0 * dx, 0.4 * dx, 2
    prims = lambda step: [(pA, None, 2, 5, 8), (pB, dB * np.float32(1.0 if step == 1 else -0.5), 1, 4, 10)]

    g = api.Grid(n, n, n, dx)
    for f in range(6):
        g.set_domain_bc(f, bc_t[f], bc_v[f])

    def loss_dev(U):
        return 0.5 * sum((a.double() ** 2).sum() for a in U), [a.clone() for a in U]
    J, grads, gU0 = ro.rollout_parametric(g, [dev(torch, a) for a in U0], prims, nsteps, dt, loss_dev, tol=1e-7,
                                          maxit=400, band=band)

    def loss_ref(U):
        return 0.5 * sum(float(np.sum(a * a)) for a in U), [a.copy() for a in U]
    p64 = lambda step: [(p.astype(np.float64), None if d is None else d.astype(np.float64), K, N, M)
                        for (p, d, K, N, M) in prims(step)]
    Jr, gr, gU0r = G.rollout_parametric(U0, p64, nsteps, dt, dx, 1.0, bc, loss_ref, band=band)
    assert abs(J - Jr) < 1e-4 * abs(Jr)
    for s in range(nsteps):
        for i in range(2):
            for got, ref in zip(grads[s][i], gr[s][i]):
                assert (got is None) == (ref is None)
                if ref is not None:
                    assert np.max(np.abs(ref)) > 0
                    assert np.max(np.abs(got - ref)) < 1e-3 * np.max(np.abs(ref)), (s, i)
    num = np.sqrt(sum(float(((a.cpu().numpy() - b) ** 2).sum()) for a, b in zip(gU0, gU0r)))
    assert num < 1e-3 * np.sqrt(sum(float((b ** 2).sum()) for b in gU0r))
    g.close()
