"""Pins for the oracle's quadratic B-spline basis (reading A20):
what the mathematics of the quadratic B-spline fixes, independent of the oracle's code.  CPU only.

N(u) = 3/4 - u^2 (|u| < 1/2), (3/2 - |u|)^2 / 2 (1/2 <= |u| < 3/2), 0 otherwise; phi_i(X) = prod_a N((X_a - x_{i,a}) / h).
"""
import numpy as np
import pytest


def _cfg(dim, n, **kw):
    c = dict(dim=dim, n=list(n), dx=1.0 / n[0], gamma=1.4, c0=1.0, c1=1.0, visc_form=0, bc=[[0, 0]] * dim, basis=1)
    c.update(kw)
    return c


def _N(u):
    u = np.abs(u)
    return np.where(u < 0.5, 0.75 - u * u, np.where(u < 1.5, 0.5 * (1.5 - u) ** 2, 0.0))


def _dN(u):
    a = np.abs(u)
    return np.where(a < 0.5, -2.0 * u, np.where(a < 1.5, -np.sign(u) * (1.5 - a), 0.0))


def _node_coords(o, h):
    idx = np.arange(o.num_nodes)
    nn = o.nn
    return np.stack([idx % nn[0], (idx // nn[0]) % nn[1], idx // (nn[0] * nn[1])])[: o.dim] * h


def _global_splines(o, cfg, x):
    """phi_i(X_k), grad phi_i(X_k) for ALL (node, particle) pairs from the global definition, periodic distance."""
    dim, h = cfg["dim"], cfg["dx"]
    xn = _node_coords(o, h)
    Nn, N = xn.shape[1], x.shape[1]
    w1, g1 = np.ones((dim, Nn, N)), np.zeros((dim, Nn, N))
    for a in range(dim):
        La = cfg["n"][a] * h
        d = x[a][None, :] - xn[a][:, None]
        d = d - La * np.rint(d / La)
        w1[a] = _N(d / h)
        g1[a] = _dN(d / h) / h
    phi = np.prod(w1, axis=0)
    grad = np.zeros((dim, Nn, N))
    for a in range(dim):
        grad[a] = g1[a] * np.prod(np.delete(w1, a, axis=0), axis=0)
    return phi, grad


def _particles(rng, cfg, N):
    dim, h = cfg["dim"], cfg["dx"]
    L = np.array(cfg["n"][:dim]) * h
    x = rng.uniform(0, 1, (dim, N)) * L[:, None]
    v = 0.3 * rng.standard_normal((dim, N))
    rho = rng.uniform(0.5, 2.0, N)
    return x, v, rho * h ** dim * rng.uniform(0.2, 0.3, N), rho, rng.uniform(1.0, 3.0, N), rng.uniform(0.0, 0.2, N)


def test_quadratic_weights_closed_form(po):
    """One particle at X/h = (2.25, 4.5): x: base node 1, f = 1.25 -> 1/32, 11/16, 9/32; y: base 4, f = 1/2 -> 1/2, 1/2, 0."""
    cfg = _cfg(2, [8, 8])
    o = po.Oracle(cfg)
    h = cfg["dx"]
    node, phi, grad = o.shape_quadratic(np.array([2.25 * h, 4.5 * h]))
    wx, wy = np.array([1 / 32, 11 / 16, 9 / 32]), np.array([0.5, 0.5, 0.0])
    np.testing.assert_allclose(phi.reshape(3, 3), np.outer(wy, wx), rtol=0, atol=1e-16)
    np.testing.assert_array_equal(node.reshape(3, 3), (np.arange(4, 7)[:, None] * 8 + np.arange(1, 4)[None, :]))
    gx, gy = np.array([-0.25, -0.5, 0.75]) / h, np.array([-1.0, 1.0, 0.0]) / h
    np.testing.assert_allclose(grad[:, 0].reshape(3, 3), np.outer(wy, gx), rtol=1e-15, atol=1e-14)
    np.testing.assert_allclose(grad[:, 1].reshape(3, 3), np.outer(gy, wx), rtol=1e-15, atol=1e-14)


@pytest.mark.parametrize("dim", [2, 3])
def test_quadratic_moments(po, dim):
    """sum phi = 1, sum grad phi = 0, sum phi (x_i - X) = 0, and the spline's second moment sum phi (x_i - X)_a^2 = h^2 / 4
    (what distinguishes the quadratic B-spline from every other 3-node partition of unity); periodic wrap included."""
    n = [6, 5, 7][:dim]
    cfg = _cfg(dim, n, dx=0.2)
    o = po.Oracle(cfg)
    h = cfg["dx"]
    xn = _node_coords(o, h)
    L = np.array(n) * h
    rng = np.random.default_rng(11)
    pts = list(rng.uniform(0, 1, (40, dim)) * L) + [np.zeros(dim), L * (1 - 1e-16), 0.5 * h * np.ones(dim), 1.5 * h * np.ones(dim)]
    for X in pts:
        node, phi, grad = o.shape_quadratic(np.asarray(X, dtype=float))
        assert len(set(node.tolist())) == 3 ** dim and (phi >= 0).all()
        assert abs(phi.sum() - 1.0) < 1e-15
        np.testing.assert_allclose(grad.sum(axis=0), 0.0, atol=1e-13 / h)
        d = xn[:, node] - np.asarray(X)[:, None]
        d = d - L[:, None] * np.rint(d / L[:, None])
        np.testing.assert_allclose((phi * d).sum(axis=1), 0.0, atol=1e-15)
        np.testing.assert_allclose((phi * d * d).sum(axis=1), 0.25 * h * h, rtol=1e-13)
        # gradient reproduces a linear field: sum_i grad_a phi_i (x_i - X)_b = delta_ab
        np.testing.assert_allclose(grad.T @ d.T, np.eye(dim), atol=1e-13)


def test_quadratic_gradient_is_continuous_where_q1_jumps(po):
    """C^1: crossing a cell face or a cell centre changes neither phi nor grad phi of any node (the Q1 gradient jumps at a
    face: the cell-crossing noise the paper discusses)."""
    cfg = _cfg(2, [8, 8])
    o = po.Oracle(cfg)
    h, eps = cfg["dx"], 1e-9
    for s in (3.0, 3.5):                   # a face and a cell centre (where the base node of the support changes)
        vals = []
        for sx in (s - eps, s + eps):
            node, phi, grad = o.shape_quadratic(np.array([sx * h, 2.3 * h]))
            full_p, full_g = np.zeros(o.num_nodes), np.zeros((o.num_nodes, 2))
            full_p[node], full_g[node] = phi, grad
            vals.append((full_p, full_g))
        assert np.abs(vals[0][0] - vals[1][0]).max() < 4 * eps
        assert np.abs(vals[0][1] - vals[1][1]).max() * h < 8 * eps
    q1 = po.Oracle(_cfg(2, [8, 8], basis=0))
    ga = q1.shape(np.array([(3.0 - eps) * h, 2.3 * h]))
    gb = q1.shape(np.array([(3.0 + eps) * h, 2.3 * h]))
    fa, fb = np.zeros((q1.num_nodes, 2)), np.zeros((q1.num_nodes, 2))
    fa[ga[0]], fb[gb[0]] = ga[2], gb[2]
    assert np.abs(fa - fb).max() * h > 0.5


@pytest.mark.parametrize("dim", [2, 3])
def test_quadratic_step_against_brute_force(po, dim):
    """Every line of Algorithm 1 that maps between particles and grid, with the 3^d-node code of the oracle against the
    global definition summed over ALL (particle, node) pairs (eqs. 16-19)."""
    n = [7, 6, 5][:dim]
    cfg = _cfg(dim, n, dx=1.0 / 7)
    o = po.Oracle(cfg)
    rng = np.random.default_rng(5 + dim)
    x, v, mass, rho, e, q = _particles(rng, cfg, 150)
    o.load_particles(x, v, mass, rho, e, q)
    phi, grad = _global_splines(o, cfg, x)
    dt = 2e-3
    o.grid_reset(); o.p2g1()
    S = ((cfg["gamma"] - 1.0) * rho * e + q) * mass / rho
    m = phi @ mass
    np.testing.assert_allclose(o.grid(po.G_MASS), m, rtol=1e-13)
    np.testing.assert_allclose(o.grid(po.G_MOM), np.stack([phi @ (mass * v[a]) for a in range(dim)]), rtol=1e-12, atol=1e-17)
    f = np.stack([grad[a] @ S for a in range(dim)])
    np.testing.assert_allclose(o.grid(po.G_FORCE), f, rtol=1e-11, atol=1e-12 * np.abs(f).max())
    o.grid_bc(); o.grid_advance(dt); o.g2p_velocity(dt)
    mvp = np.stack([phi @ (mass * v[a]) for a in range(dim)]) + dt * f
    np.testing.assert_allclose(o.particles(po.P_VBAR), np.stack([(mvp[a] / m) @ phi for a in range(dim)]), rtol=1e-11)
    acc = np.stack([(f[a] / m) @ phi for a in range(dim)])
    np.testing.assert_allclose(o.particles(po.P_ACC), acc, rtol=1e-10, atol=1e-11 * np.abs(acc).max())
    vp = v + dt * acc
    np.testing.assert_allclose(o.particles(po.P_V), vp, rtol=1e-12)
    o.p2g2(); o.grid_bc2()
    mv2 = np.stack([phi @ (mass * vp[a]) for a in range(dim)])
    np.testing.assert_allclose(o.grid(po.G_MOM2), mv2, rtol=1e-12, atol=1e-17)
    o.particle_update(dt)
    D = sum((mv2[a] / m) @ grad[a] for a in range(dim))
    np.testing.assert_allclose(o.particles(po.P_DIV), D, rtol=1e-9, atol=1e-10 * np.abs(D).max())
    np.testing.assert_allclose(o.particles(po.P_RHO), rho / (1.0 + dt * D), rtol=1e-12)


@pytest.mark.parametrize("dim", [2, 3])
def test_quadratic_conservation_periodic(po, dim):
    """The conservation statements of the Q1 pins hold for any partition of unity: mass, momentum, sum f = 0, and the
    discrete work identity sum M (E' - E) = -dt sum_i f_i . (mv2_i / m_i)."""
    n = [8, 7, 6][:dim]
    cfg = _cfg(dim, n, dx=1.0 / 8)
    o = po.Oracle(cfg)
    rng = np.random.default_rng(21)
    x, v, mass, rho, e, q = _particles(rng, cfg, 900)
    o.load_particles(x, v, mass, rho, e, q)
    dt = 1e-3
    o.grid_reset(); o.p2g1()
    assert abs(o.grid(po.G_MASS).sum() - mass.sum()) <= 1e-13 * mass.sum()
    mom = (mass * v).sum(axis=1)
    np.testing.assert_allclose(o.grid(po.G_MOM).sum(axis=1), mom, atol=1e-13 * np.abs(mass * v).sum())
    f = o.grid(po.G_FORCE).copy()
    m = o.grid(po.G_MASS).copy()
    assert np.abs(f.sum(axis=1)).max() <= 1e-12 * np.abs(f).sum()
    o.grid_bc(); o.grid_advance(dt); o.g2p_velocity(dt)
    np.testing.assert_allclose((mass * o.particles(po.P_V)).sum(axis=1), mom + dt * f.sum(axis=1), atol=1e-13 * np.abs(mass * v).sum())
    o.p2g2(); o.grid_bc2()
    mv2 = o.grid(po.G_MOM2).copy()
    o.particle_update(dt)
    work = -dt * (f * mv2 / m).sum()
    dE = (mass * (o.particles(po.P_E) - e)).sum()
    # Q of this step (reading A2) enters the energy update but not this step's force: take its share out
    D = o.particles(po.P_DIV); Qn = o.particles(po.P_Q)
    dE_p = dE + dt * (mass * (Qn - q) / rho * D).sum()
    assert abs(dE_p - work) <= 1e-11 * max(abs(work), np.abs(mass * e).sum() * dt)


def test_quadratic_needs_a_periodic_grid(po):
    with pytest.raises(ValueError):
        po.Oracle(_cfg(2, [8, 8], bc=[[1, 1], [0, 0]]))
    with pytest.raises(ValueError):
        po.Oracle(_cfg(2, [2, 8]))
