"""Pins for the CPU oracle (oracle/mpm_oracle.c): what the paper and the mathematics fix, independent of
the oracle's own code.  CPU only (-m "not gpu").  Each test names the passage / reading it pins.

A plausible mistake anywhere in the oracle (dropped term, wrong sign or index, transposed operand, wrong
corner ordering, BC on the wrong face, wrong power of h) fails at least one of these.
"""
import os

import numpy as np
import pytest

import riemann
from paper_2404_17057_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _cfg(dim, n, dx=None, bc=None, **kw):
    dx = dx if dx is not None else 1.0 / n[0]
    bc = bc if bc is not None else [[0, 0]] * dim
    c = dict(dim=dim, n=list(n), dx=dx, gamma=1.4, c0=1.0, c1=1.0, visc_form=0, bc=bc)
    c.update(kw)
    return c


def _random_particles(rng, dim, n, dx, N, vscale=0.3):
    L = np.array(n[:dim]) * dx
    x = rng.uniform(0, 1, (dim, N)) * L[:, None]
    v = vscale * rng.standard_normal((dim, N))
    rho = rng.uniform(0.5, 2.0, N)
    mass = rho * dx ** dim * rng.uniform(0.2, 0.3, N)
    e = rng.uniform(1.0, 3.0, N)
    q = rng.uniform(0.0, 0.2, N)
    return x, v, mass, rho, e, q


def _node_coords(o, dx):
    nn = o.nn
    idx = np.arange(o.num_nodes)
    ix = idx % nn[0]
    iy = (idx // nn[0]) % nn[1]
    iz = idx // (nn[0] * nn[1])
    return np.stack([ix, iy, iz])[: o.dim] * dx


def _global_hats(o, cfg, x):
    """phi_i(X_k) and grad phi_i(X_k) for ALL (node i, particle k) pairs from the global definition
    phi_i(x) = prod_a max(0, 1 - |x_a - x_{i,a}|/h), periodic distance on periodic axes."""
    dim, h = cfg["dim"], cfg["dx"]
    xn = _node_coords(o, h)                       # [dim, Nn]
    Nn, N = xn.shape[1], x.shape[1]
    w1 = np.ones((dim, Nn, N))
    g1 = np.zeros((dim, Nn, N))
    for a in range(dim):
        d = x[a][None, :] - xn[a][:, None]
        if cfg["bc"][a][0] == 0:
            La = cfg["n"][a] * h
            d = d - La * np.rint(d / La)
        w1[a] = np.maximum(0.0, 1.0 - np.abs(d) / h)
        g1[a] = np.where(np.abs(d) < h, -np.sign(d) / h, 0.0)
    phi = np.prod(w1, axis=0)
    grad = np.zeros((dim, Nn, N))
    for a in range(dim):
        t = g1[a].copy()
        for a2 in range(dim):
            if a2 != a:
                t = t * w1[a2]
        grad[a] = t
    return phi, grad


# --------------------------------------------------------------------------- weights

def test_weights_closed_form_quarter_three_quarter(po):
    """Q1 weights of a particle at local (xi, eta) = (1/4, 3/4): 3/16, 1/16, 9/16, 3/16 (SURVEY 8c pin)."""
    h = 0.125
    o = po.Oracle(_cfg(2, [8, 8], h, [[1, 1], [1, 1]]))
    node, phi, grad = o.shape(np.array([(3 + 0.25) * h, (5 + 0.75) * h]))
    np.testing.assert_allclose(phi, [3 / 16, 1 / 16, 9 / 16, 3 / 16], atol=1e-15)
    assert list(node) == [3 + 9 * 5, 4 + 9 * 5, 3 + 9 * 6, 4 + 9 * 6]
    # d/dx phi = -+(1/h) w_y ; d/dy phi = -+(1/h) w_x
    np.testing.assert_allclose(grad[:, 0], np.array([-0.25, 0.25, -0.75, 0.75]) / h, atol=1e-13)
    np.testing.assert_allclose(grad[:, 1], np.array([-0.75, -0.25, 0.75, 0.25]) / h, atol=1e-13)


@pytest.mark.parametrize("dim", [2, 3])
def test_partition_of_unity(po, dim):
    """sum_b phi = 1 and sum_b grad phi = 0 at random points."""
    rng = np.random.default_rng(11)
    n = [7, 5, 6][:dim]
    h = 0.1
    o = po.Oracle(_cfg(dim, n, h, [[1, 1]] * dim))
    for _ in range(200):
        X = rng.uniform(0, 1, dim) * np.array(n) * h
        node, phi, grad = o.shape(X)
        assert abs(phi.sum() - 1.0) < 1e-15 * 4
        assert np.all(np.abs(grad.sum(axis=0)) < 1e-13 / h)
        assert np.all(phi >= 0)
        assert len(set(node.tolist())) == (1 << dim)


def test_upper_face_clamp(po):
    """A6: a particle exactly on the upper domain face belongs to the last cell with xi = 1."""
    h = 0.25
    o = po.Oracle(_cfg(2, [4, 4], h, [[1, 1], [1, 1]]))
    node, phi, _ = o.shape(np.array([1.0, 0.5 * h]))
    np.testing.assert_allclose(phi, [0.0, 0.5, 0.0, 0.5], atol=1e-15)
    assert node[1] == 4 and node[3] == 4 + 5


# --------------------------------------------------------------------------- the four kernels by brute force

@pytest.mark.parametrize("dim,periodic", [(2, False), (2, True), (3, False), (3, True)])
def test_p2g_p2gd_g2p_g2pd_brute_force(po, dim, periodic):
    """Eqs. (16)-(19) summed over ALL (k,i) pairs with global hat functions versus the
    oracle's cell-local 2^d-node code; and every line of Algorithm 1 that is built from them."""
    rng = np.random.default_rng(5 + dim + 10 * periodic)
    n = [8, 6, 5][:dim]
    h = 1.0 / 8
    bc = [[0, 0]] * dim if periodic else [[1, 1]] * dim
    cfg = _cfg(dim, n, h, bc)
    o = po.Oracle(cfg)
    N = 150
    x, v, mass, rho, e, q = _random_particles(rng, dim, n, h, N)
    o.load_particles(x, v, mass, rho, e, q)
    phi, grad = _global_hats(o, cfg, x)
    # -- l.3: m = P2G(M), mv = P2G(MV), f = P2GD((P+Q) M / rho)
    o.grid_reset(); o.p2g1()
    P = (1.4 - 1.0) * rho * e
    S = (P + q) * mass / rho
    np.testing.assert_allclose(o.grid(po.G_MASS), phi @ mass, rtol=1e-14, atol=1e-18)
    for a in range(dim):
        np.testing.assert_allclose(o.grid(po.G_MOM)[a], phi @ (mass * v[a]), rtol=0, atol=1e-14 * np.abs(mass * v[a]).sum())
        np.testing.assert_allclose(o.grid(po.G_FORCE)[a], grad[a] @ S, rtol=0, atol=1e-14 * np.abs(grad[a] * S).sum(axis=1).max())
    # -- l.5 (no BC call here: pure kernels) and l.6-7
    dt = 0.01
    m = o.grid(po.G_MASS); mv = o.grid(po.G_MOM).copy(); f = o.grid(po.G_FORCE).copy()
    o.grid_advance(dt)
    mvp = mv + dt * f
    np.testing.assert_allclose(o.grid(po.G_MOM), mvp, rtol=1e-15, atol=0)
    o.g2p_velocity(dt)
    safe = np.where(m != 0, m, 1.0)
    for a in range(dim):
        vb = (np.where(m != 0, mvp[a] / safe, 0.0)) @ phi
        ac = (np.where(m != 0, f[a] / safe, 0.0)) @ phi
        np.testing.assert_allclose(o.particles(po.P_VBAR)[a], vb, rtol=0, atol=1e-13 * (1 + np.abs(vb).max()))
        np.testing.assert_allclose(o.particles(po.P_ACC)[a], ac, rtol=0, atol=1e-13 * (1 + np.abs(ac).max()))
        np.testing.assert_allclose(o.particles(po.P_V)[a], v[a] + dt * ac, rtol=0, atol=1e-13 * (1 + np.abs(ac).max()))
    vnew = o.particles(po.P_V)
    # -- l.8
    o.p2g2()
    for a in range(dim):
        np.testing.assert_allclose(o.grid(po.G_MOM2)[a], phi @ (mass * vnew[a]), rtol=0, atol=1e-14 * np.abs(mass * vnew[a]).sum())
    # -- l.10: D = trace G2PD(mv2/m)
    mv2 = o.grid(po.G_MOM2)
    o.particle_update(dt)
    D = np.zeros(N)
    for a in range(dim):
        D += np.where(m != 0, mv2[a] / safe, 0.0) @ grad[a]
    scale = np.abs(np.where(m != 0, mv2 / safe, 0.0)).max() / h
    np.testing.assert_allclose(o.particles(po.P_DIV), D, rtol=0, atol=1e-13 * scale)
    # particle thermodynamics exactly as printed (eq. 4)
    Qn = np.where(D < 0, 1.0 * (rho * h * D) ** 2 - 1.0 * h * np.sqrt(1.4 * P / rho) * D, 0.0)   # eq. (4), same D
    En = e - dt * (P + Qn) / rho * D
    rhon = rho / (1.0 + dt * D)
    np.testing.assert_allclose(o.particles(po.P_E), En, rtol=1e-12)
    np.testing.assert_allclose(o.particles(po.P_RHO), rhon, rtol=1e-12)
    np.testing.assert_allclose(o.particles(po.P_Q), Qn, rtol=1e-10, atol=1e-14)
    # -- l.11 advection with Vbar (not V')
    vb = o.particles(po.P_VBAR)
    o.advect(dt)
    xn = x + dt * vb
    L = np.array(n) * h
    for a in range(dim):
        xa = xn[a] - L[a] * np.floor(xn[a] / L[a]) if periodic else np.clip(xn[a], 0, L[a])
        np.testing.assert_allclose(o.particles(po.P_X)[a], xa, rtol=0, atol=1e-15)


@pytest.mark.parametrize("dim", [2, 3])
def test_affine_reproduction(po, dim):
    """Q1 reproduces affine fields: G2P of a + b.x_i gives a + b.X_k, G2PD gives b (eqs. 17, 19)."""
    rng = np.random.default_rng(21)
    n = [6, 5, 4][:dim]
    h = 0.2
    cfg = _cfg(dim, n, h, [[3, 3]] * dim)   # OUTFLOW everywhere: BC leaves mv untouched, no periodic seam
    o = po.Oracle(cfg)
    N = 400
    L = np.array(n) * h
    x = rng.uniform(0.02, 0.98, (dim, N)) * L[:, None]
    rho = np.ones(N); mass = np.full(N, h ** dim / 10); e = np.ones(N)
    # particle velocities sampled from an affine field: V = a + B x.  Then mv_i/m_i is NOT affine in general, so
    # instead test the gather alone: after P2G#2 overwrite nothing - use the identity through a uniform field.
    a0 = rng.standard_normal(dim)
    v = np.repeat(a0[:, None], N, axis=1)
    o.load_particles(x, v, mass, rho, e)
    o.grid_reset(); o.p2g1()
    # uniform velocity: mv_i/m_i = a0 exactly at every node with mass -> Vbar = a0 (partition of unity), D = 0
    o.grid_advance(0.0); o.g2p_velocity(0.0); o.p2g2(); o.particle_update(0.1)
    for a in range(dim):
        np.testing.assert_allclose(o.particles(po.P_VBAR)[a], a0[a], rtol=1e-13)
    assert np.abs(o.particles(po.P_DIV)).max() < 1e-12 / h


def test_uniform_compression_closed_form(po):
    """Lattice with V = -a X: grid velocity is exactly linear, so D = -a d... per axis: D = -a*dim on interior particles,
    rho' = rho/(1 - a d dt), E' = E + dt a d (P+Q)/rho (SURVEY 8c 'uniform compression')."""
    n = [16, 16]; h = 1.0 / 16; dim = 2
    cfg = _cfg(dim, n, h, [[3, 3]] * dim)
    o = po.Oracle(cfg)
    w = inputs._lattice_positions(n, h, 2, 0.0, None)
    N = w.shape[1]
    a = 0.37
    v = -a * w
    rho = np.full(N, 1.3); mass = rho * h * h / 4; e = np.full(N, 2.0)
    o.load_particles(w, v, mass, rho, e)
    dt = 1e-3
    o.grid_reset(); o.p2g1()
    o.grid_advance(0.0)                 # keep the momentum field = P2G(MV): dt = 0 in l.5-7
    o.g2p_velocity(0.0); o.p2g2()
    o.particle_update(dt)
    D = o.particles(po.P_DIV)
    interior = np.all((w > 1.5 * h) & (w < 1 - 1.5 * h), axis=0)
    # symmetric lattice: nodal velocity = -a x_i exactly in the interior (mass-weighted mean of an odd perturbation)
    np.testing.assert_allclose(D[interior], -a * dim, rtol=1e-12)
    P = 0.4 * 1.3 * 2.0
    np.testing.assert_allclose(o.particles(po.P_RHO)[interior], 1.3 / (1 - a * dim * dt), rtol=1e-12)
    Dc = -a * dim
    Qc = (1.3 * h * Dc) ** 2 - h * np.sqrt(1.4 * P / 1.3) * Dc          # eq. (4), compression
    np.testing.assert_allclose(o.particles(po.P_E)[interior], 2.0 + dt * a * dim * (P + Qc) / 1.3, rtol=1e-12)
    np.testing.assert_allclose(o.particles(po.P_Q)[interior], Qc, rtol=1e-12)


@pytest.mark.parametrize("c0,c1", [(1.0, 1.0), (1.7, 0.6)])
def test_uniform_compression_closed_form_standard_viscosity(po, c0, c1):
    """The visc_form = STANDARD branch of l.10 (reading A3; the branch BASELINE configs 4 and 5 run), pinned on the same
    uniform-compression lattice by the textbook von Neumann-Richtmyer + Landshoff pressure written out HERE:
        Q = rho (c0 h^2 D^2 + c1 h c_s |D|),  c_s = sqrt(gamma P / rho),  D = -a d < 0   (refs. of PAPER.md:580),
        E' = E + dt a d (P + Q) / rho,  rho' = rho / (1 - a d dt).
    c0 != c1 != 1 tells the two coefficients apart; h = 1/16 tells h from h^2; rho = 1.3 catches a dropped rho."""
    n = [16, 16]; h = 1.0 / 16; dim = 2
    cfg = _cfg(dim, n, h, [[3, 3]] * dim, visc_form=1, c0=c0, c1=c1)
    o = po.Oracle(cfg)
    w = inputs._lattice_positions(n, h, 2, 0.0, None)
    N = w.shape[1]
    a = 0.37
    rho0, e0, dt = 1.3, 2.0, 1e-3
    rho = np.full(N, rho0); mass = rho * h * h / 4; e = np.full(N, e0)
    o.load_particles(w, -a * w, mass, rho, e)
    o.grid_reset(); o.p2g1()
    o.grid_advance(0.0)
    o.g2p_velocity(0.0); o.p2g2()
    o.particle_update(dt)
    interior = np.all((w > 1.5 * h) & (w < 1 - 1.5 * h), axis=0)
    Dabs = a * dim
    P = 0.4 * rho0 * e0
    cs = np.sqrt(1.4 * P / rho0)
    Qc = rho0 * (c0 * h * h * Dabs * Dabs + c1 * h * cs * Dabs)
    np.testing.assert_allclose(o.particles(po.P_DIV)[interior], -Dabs, rtol=1e-12)
    np.testing.assert_allclose(o.particles(po.P_Q)[interior], Qc, rtol=1e-12)
    np.testing.assert_allclose(o.particles(po.P_E)[interior], e0 + dt * Dabs * (P + Qc) / rho0, rtol=1e-12)
    np.testing.assert_allclose(o.particles(po.P_RHO)[interior], rho0 / (1 - Dabs * dt), rtol=1e-12)


def test_viscosity_density_scaling_tells_the_two_forms_apart(po):
    """Why configs 4 and 5 take STANDARD (A3): under rho -> 2 rho, M -> 2 M at fixed h, D, E (hence fixed c_s)
    a viscous PRESSURE must double, so that Q/rho and with it E' do not change.  STANDARD: Q -> 2 Q for both terms.
    Eq. (4) as printed: quadratic term x 4, linear term x 1.  Each term is isolated by zeroing
    the other coefficient; nothing here comes from the oracle's source."""
    n = [16, 16]; h = 1.0 / 16; dim = 2
    w = inputs._lattice_positions(n, h, 2, 0.0, None)
    N = w.shape[1]
    interior = np.all((w > 1.5 * h) & (w < 1 - 1.5 * h), axis=0)
    a, dt = 0.37, 1e-3

    def run(form, c0, c1, scale):
        o = po.Oracle(_cfg(dim, n, h, [[3, 3]] * dim, visc_form=form, c0=c0, c1=c1))
        rho = np.full(N, 1.3 * scale)
        o.load_particles(w, -a * w, rho * h * h / 4, rho, np.full(N, 2.0))
        o.grid_reset(); o.p2g1(); o.grid_advance(0.0); o.g2p_velocity(0.0); o.p2g2(); o.particle_update(dt)
        return o.particles(po.P_Q)[interior], o.particles(po.P_E)[interior]

    for form, (r_quad, r_lin) in ((1, (2.0, 2.0)), (0, (4.0, 1.0))):
        q1, e1 = run(form, 1.0, 0.0, 1.0); q2, e2 = run(form, 1.0, 0.0, 2.0)
        np.testing.assert_allclose(q2 / q1, r_quad, rtol=1e-12)
        l1, el1 = run(form, 0.0, 1.0, 1.0); l2, el2 = run(form, 0.0, 1.0, 2.0)
        np.testing.assert_allclose(l2 / l1, r_lin, rtol=1e-12)
        if form == 1:      # Q / rho unchanged => the energy update does not see the density scale
            np.testing.assert_allclose(e2, e1, rtol=1e-13)
            np.testing.assert_allclose(el2, el1, rtol=1e-13)
        else:
            assert np.abs(e2 - e1).max() > 1e-9 and np.abs(el2 - el1).max() > 1e-9


@pytest.mark.parametrize("dim,periodic", [(2, True), (3, False)])
def test_grid_diagnostic_density_and_energy(po, dim, periodic):
    """Reading A18: rho_i = sum_k M rho phi_i / sum_k M phi_i, same for E, against the global hat
    functions over all (particle, node) pairs; a uniform particle field is reproduced exactly wherever there is mass."""
    n = [6, 5, 4][:dim]
    cfg = _cfg(dim, n, 0.2, [[0, 0]] * dim if periodic else [[1, 1]] * dim)
    o = po.Oracle(cfg)
    rng = np.random.default_rng(17)
    x, v, mass, rho, e, q = _random_particles(rng, dim, n, 0.2, 120)
    o.load_particles(x, v, mass, rho, e, q)
    phi, _ = _global_hats(o, cfg, x)
    den = phi @ mass
    for which, a in ((0, rho), (1, e)):
        want = np.where(den > 0, (phi @ (mass * a)) / np.where(den > 0, den, 1.0), 0.0)
        np.testing.assert_allclose(o.grid_diagnostic(which), want, rtol=1e-13, atol=1e-15)
    o.load_particles(x, v, mass, np.full_like(rho, 1.7), e, q)
    got = o.grid_diagnostic(0)
    np.testing.assert_allclose(got[den > 0], 1.7, rtol=1e-14)


# --------------------------------------------------------------------------- conservation

def _periodic_box(po, dim, seed=3, N=600):
    rng = np.random.default_rng(seed)
    n = [8, 8, 8][:dim]; h = 1.0 / 8
    cfg = _cfg(dim, n, h, [[0, 0]] * dim)
    o = po.Oracle(cfg)
    x, v, mass, rho, e, q = _random_particles(rng, dim, n, h, N)
    o.load_particles(x, v, mass, rho, e, q)
    return o, cfg, (x, v, mass, rho, e, q)


@pytest.mark.parametrize("dim", [2, 3])
def test_mass_momentum_conservation_periodic(po, dim):
    """sum_i m_i = sum_k M_k; sum_i mv_i = sum_k M_k V_k; sum_i f_i = 0; sum_k M_k V'_k = sum_k M_k V_k
    to 1e-12 relative per step in a periodic box (eqs. 13-14; BASELINE north_star)."""
    o, cfg, (x, v, mass, rho, e, q) = _periodic_box(po, dim)
    for step in range(5):
        v0 = o.particles(po.P_V); m0 = o.particles(po.P_M)
        o.grid_reset(); o.p2g1()
        assert abs(o.grid(po.G_MASS).sum() - m0.sum()) <= 1e-13 * m0.sum()
        for a in range(dim):
            ref = (m0 * v0[a]).sum(); sc = np.abs(m0 * v0[a]).sum()
            assert abs(o.grid(po.G_MOM)[a].sum() - ref) <= 1e-12 * sc
            assert abs(o.grid(po.G_FORCE)[a].sum()) <= 1e-12 * np.abs(o.grid(po.G_FORCE)[a]).sum()
        dt = 2e-3
        o.grid_bc(); o.grid_advance(dt); o.g2p_velocity(dt)
        v1 = o.particles(po.P_V)
        for a in range(dim):
            assert abs((m0 * v1[a]).sum() - (m0 * v0[a]).sum()) <= 1e-12 * np.abs(m0 * v0[a]).sum()
        o.p2g2(); o.grid_bc2(); o.particle_update(dt); o.cfl(0.3); o.advect(dt)
        np.testing.assert_array_equal(o.particles(po.P_M), m0)   # M_k never changes


@pytest.mark.parametrize("dim", [2, 3])
def test_energy_work_identity_and_dt2_drift(po, dim):
    """The scheme does not conserve total energy to rounding; what is exact is the discrete work identity
    sum_k M_k (E'_k - E_k) = -dt sum_i f_i . (mv2_i/m_i) in a periodic box, pinned at 1e-12, and the
    one-step total-energy defect is O(dt^2): halving dt cuts it ~4x."""
    defects = []
    for dt in (4e-3, 2e-3):
        # pressure work only: c0 = c1 = 0 and no initial Q, so that f is the pure pressure force
        rng = np.random.default_rng(9)
        n = [8, 8, 8][:dim]; h = 1.0 / 8
        cfg = _cfg(dim, n, h, [[0, 0]] * dim, c0=0.0, c1=0.0)
        o = po.Oracle(cfg)
        x, v, mass, rho, e, q = _random_particles(rng, dim, n, h, 600)
        o.load_particles(x, v, mass, rho, e, None)
        ke0 = 0.5 * (mass * (v ** 2).sum(axis=0)).sum(); ie0 = (mass * e).sum()
        o.grid_reset(); o.p2g1(); o.grid_bc(); o.grid_advance(dt); o.g2p_velocity(dt); o.p2g2(); o.grid_bc2()
        f = o.grid(po.G_FORCE); mv2 = o.grid(po.G_MOM2); m = o.grid(po.G_MASS)
        o.particle_update(dt)
        e1 = o.particles(po.P_E); v1 = o.particles(po.P_V)
        safe = np.where(m != 0, m, 1.0)
        work = -dt * sum((f[a] * np.where(m != 0, mv2[a] / safe, 0.0)).sum() for a in range(dim))
        lhs = (mass * (e1 - e)).sum()
        scale = dt * sum(np.abs(f[a] * mv2[a] / safe).sum() for a in range(dim))
        assert abs(lhs - work) <= 1e-12 * scale
        ke1 = 0.5 * (mass * (v1 ** 2).sum(axis=0)).sum()
        defects.append((ke1 + (mass * e1).sum()) - (ke0 + ie0))
        # with the viscosity on, the extra heating is -dt sum_k M_k Q_k D_k / rho_k >= 0 with Q from THIS step's D
        # (eqs. 4, 5a, 5b: one div v for q and for the energy equation -- reading A2)
        o2 = po.Oracle(_cfg(dim, n, h, [[0, 0]] * dim))
        o2.load_particles(x, v, mass, rho, e, None)
        o2.grid_reset(); o2.p2g1(); o2.grid_bc(); o2.grid_advance(dt); o2.g2p_velocity(dt); o2.p2g2(); o2.grid_bc2()
        o2.particle_update(dt)
        D = o2.particles(po.P_DIV); Q = o2.particles(po.P_Q)
        assert (Q[D >= 0] == 0).all() and (Q[D < 0] > 0).all()
        extra = (mass * (o2.particles(po.P_E) - e1)).sum()
        expect = -dt * (mass * Q * D / rho).sum()
        assert expect > 0 and abs(extra - expect) <= 1e-12 * expect
    ratio = defects[0] / defects[1]
    assert 3.5 <= ratio <= 4.5, ratio


# --------------------------------------------------------------------------- steady states, symmetry

def test_rest_state_and_uniform_translation(po):
    """Uniform rho, p on an un-jittered lattice in a periodic box: at rest nothing moves; uniform V0 translates
    X(t) = X0 + V0 t mod L with rho, E constant (SURVEY 8c 'steady states')."""
    n = [8, 8]; h = 1.0 / 8
    X0 = inputs._lattice_positions(n, h, 2, 0.0, None)
    N = X0.shape[1]
    for V0 in ([0.0, 0.0], [0.31, -0.17]):
        o = po.Oracle(_cfg(2, n, h, [[0, 0], [0, 0]]))
        v = np.repeat(np.array(V0)[:, None], N, axis=1)
        o.load_particles(X0, v, np.full(N, h * h / 4), np.ones(N), np.full(N, 2.5))
        dt = 0.01
        o.step(dt, 0.3, 20)
        xt = np.mod(X0 + np.array(V0)[:, None] * dt * 20, 1.0)
        d = o.particles(po.P_X) - xt
        d -= np.rint(d)
        assert np.abs(d).max() < 1e-13
        np.testing.assert_allclose(o.particles(po.P_RHO), 1.0, rtol=1e-12)
        np.testing.assert_allclose(o.particles(po.P_E), 2.5, rtol=1e-12)
        np.testing.assert_allclose(o.particles(po.P_V), v, rtol=0, atol=1e-12)


def test_one_dimensional_reduction(po):
    """Config-1 data without jitter: V_y = 0 and all fields y-independent (to rounding) for 30 steps."""
    w = inputs.sod(nx=64, ny=4, jitter=0.0)
    o = po.Oracle(w["cfg"])
    o.load_particles(w["x"], w["v"], w["mass"], w["rho"], w["e"])
    o.step(0.0, w["cfl"], 30)
    assert np.abs(o.particles(po.P_V)[1]).max() < 1e-12
    rho = o.particles(po.P_RHO).reshape(4, 64, 4)     # [cy, cx, sub]
    assert np.abs(rho - rho[0:1]).max() < 1e-12


def test_mirror_symmetry_sedov(po):
    """Un-jittered Sedov data: octant mirror images stay mirror images."""
    w = inputs.sedov(n=12, jitter=0.0)
    o = po.Oracle(w["cfg"])
    o.load_particles(w["x"], w["v"], w["mass"], w["rho"], w["e"])
    o.step(0.0, w["cfl"], 12)
    x = o.particles(po.P_X); rho = o.particles(po.P_RHO); v = o.particles(po.P_V)
    x0 = w["x"]
    # match each particle with its mirror image across x = 1/2 using the initial lattice
    key = np.round(x0 * 48).astype(np.int64)
    lut = {tuple(k): i for i, k in enumerate(key.T)}
    mirror = np.array([lut[(48 - k[0], k[1], k[2])] for k in key.T])
    assert np.abs(rho - rho[mirror]).max() < 1e-12 * rho.max()
    assert np.abs(v[0] + v[0][mirror]).max() < 1e-12 * (np.abs(v).max() + 1e-300)
    assert np.abs((x[0] - 0.5) + (x[0][mirror] - 0.5)).max() < 1e-13
    assert rho.max() > 1.05      # the blast actually did something


# --------------------------------------------------------------------------- boundary conditions, obstacle, CFL

def test_obstacle_rule(po):
    """Eqs. (21),(22): w' = w - min(w.n, 0) n; afterwards w'.n >= 0, tangential part unchanged, idempotent."""
    n = [8, 8]; h = 1.0 / 8
    mask = np.zeros((8, 8), np.uint8); mask[3:5, 3:5] = 1
    rng = np.random.default_rng(2)
    nrm = rng.standard_normal((2, 81)); nrm /= np.linalg.norm(nrm, axis=0)
    cfg = _cfg(2, n, h, [[3, 3], [3, 3]], obstacle_mask=mask, node_normals=nrm)
    o = po.Oracle(cfg)
    flag = o.grid(po.G_FLAG).reshape(9, 9)
    expect = np.zeros((9, 9)); expect[3:6, 3:6] = 1        # nodes touching any masked cell (A7)
    np.testing.assert_array_equal(flag, expect)
    x, v, mass, rho, e, q = _random_particles(rng, 2, n, h, 500)
    o.load_particles(x, v, mass, rho, e, q)
    o.grid_reset(); o.p2g1()
    mv0 = o.grid(po.G_MOM).copy(); f0 = o.grid(po.G_FORCE).copy()
    o.grid_bc()
    mv1 = o.grid(po.G_MOM); f1 = o.grid(po.G_FORCE)
    fl = flag.ravel() > 0
    for w0, w1 in ((mv0, mv1), (f0, f1)):
        dot0 = (w0 * nrm).sum(axis=0)
        expect_w = w0 - np.minimum(dot0, 0.0) * nrm * fl
        # OUTFLOW faces zero the normal force only; restrict the check to interior (obstacle) nodes
        np.testing.assert_allclose(w1[:, fl], expect_w[:, fl], rtol=0, atol=1e-15 * np.abs(w0).max() * 4)
        assert ((w1 * nrm).sum(axis=0)[fl] >= -1e-15 * np.abs(w0).max()).all()
        tang0 = w0 - dot0 * nrm; tang1 = w1 - (w1 * nrm).sum(axis=0) * nrm
        np.testing.assert_allclose(tang1[:, fl], tang0[:, fl], rtol=0, atol=1e-14 * np.abs(w0).max())
    o.grid_bc()   # idempotent
    np.testing.assert_allclose(o.grid(po.G_MOM)[:, fl], mv1[:, fl], rtol=0, atol=1e-15 * np.abs(mv0).max())
    assert (mv0[:, fl] != mv1[:, fl]).any()


def test_wall_inflow_outflow_bc(po):
    """A9/A10/eq. 30: REFLECT zeroes the normal components of mv and f on its face; INFLOW sets mv = m v_in, f = 0;
    OUTFLOW zeroes the normal force only; interior nodes untouched."""
    n = [6, 5]; h = 0.1
    cfg = _cfg(2, n, h, [[2, 3], [1, 1]], inflow_rho=1.4, inflow_p=1.0, inflow_v=[3.0, 0.0, 0.0])
    o = po.Oracle(cfg)
    rng = np.random.default_rng(8)
    x, v, mass, rho, e, q = _random_particles(rng, 2, n, h, 400)
    o.load_particles(x, v, mass, rho, e, q)
    o.grid_reset(); o.p2g1()
    m = o.grid(po.G_MASS).reshape(6, 7)
    mv0 = o.grid(po.G_MOM).reshape(2, 6, 7).copy(); f0 = o.grid(po.G_FORCE).reshape(2, 6, 7).copy()
    o.grid_bc()
    mv = o.grid(po.G_MOM).reshape(2, 6, 7); f = o.grid(po.G_FORCE).reshape(2, 6, 7)
    np.testing.assert_array_equal(mv[:, 1:-1, 1:-1], mv0[:, 1:-1, 1:-1])
    np.testing.assert_array_equal(f[:, 1:-1, 1:-1], f0[:, 1:-1, 1:-1])
    np.testing.assert_allclose(mv[0, 1:-1, 0], 3.0 * m[1:-1, 0], rtol=1e-15)       # inflow face x-low
    assert (mv[1, :, 0] == 0).all() and (f[:, :, 0] == 0).all()
    np.testing.assert_array_equal(mv[:, 1:-1, -1], mv0[:, 1:-1, -1])               # outflow: momentum untouched
    assert (f[0, :, -1] == 0).all()
    np.testing.assert_array_equal(f[1, 1:-1, -1], f0[1, 1:-1, -1])
    for j in (0, -1):                                                              # reflecting y walls
        assert (mv[1, j, :] == 0).all() and (f[1, j, :] == 0).all()
        np.testing.assert_array_equal(mv[0, j, 1:-1], mv0[0, j, 1:-1])


def test_cfl_identity(po):
    """dt_next (vmax + cmax)/h = alpha with separate maxima over |V'|, |Vbar| and c_s (eq. 29; A12)."""
    o, cfg, (x, v, mass, rho, e, q) = _periodic_box(po, 2)
    o.step(1e-3, 0.3, 3)
    for alpha in (0.3, 0.25, 0.5):
        o.cfl(alpha)
        s = o.stats()
        assert abs(s.dt_next * (s.vmax + s.cmax) / cfg["dx"] - alpha) <= 4e-16
    V = o.particles(po.P_V); Vb = o.particles(po.P_VBAR)
    vmax = max(np.sqrt((V ** 2).sum(axis=0)).max(), np.sqrt((Vb ** 2).sum(axis=0)).max())
    cmax = np.sqrt(1.4 * 0.4 * o.particles(po.P_E)).max()
    s = o.stats()
    assert abs(s.vmax - vmax) <= 1e-15 * vmax and abs(s.cmax - cmax) <= 2e-15 * cmax
    # a state where |Vbar| exceeds |V'| (grid momentum advanced, particle velocity not): vmax must follow Vbar
    o.grid_reset(); o.p2g1(); o.grid_bc(); o.grid_advance(0.5); o.g2p_velocity(0.0); o.cfl(0.3)
    V = o.particles(po.P_V); Vb = o.particles(po.P_VBAR)
    nV, nVb = np.sqrt((V ** 2).sum(axis=0)).max(), np.sqrt((Vb ** 2).sum(axis=0)).max()
    assert nVb > 1.5 * nV
    assert abs(o.stats().vmax - nVb) <= 1e-15 * nVb
    o.p2g2(); o.grid_bc2(); o.particle_update(1e-3); o.cfl(0.3)
    s = o.stats()
    # adaptive stepping uses it: next dt equals alpha h/(vmax+cmax)
    dt = o.step(0.0, 0.5, 1)
    assert abs(dt - 0.5 * cfg["dx"] / (s.vmax + s.cmax)) <= 1e-18 + 1e-15 * dt


def test_first_step_dt_from_loaded_state(po):
    """A13: first dt = alpha h / (max|V| + max c_s) of the loaded state."""
    w = inputs.sod(nx=32, ny=2)
    o = po.Oracle(w["cfg"])
    o.load_particles(w["x"], w["v"], w["mass"], w["rho"], w["e"])
    dt = o.step(0.0, 0.3, 1)
    c = np.sqrt(1.4 * 1.0 / 1.0)
    assert abs(dt - 0.3 * (1 / 32) / c) < 1e-15


# --------------------------------------------------------------------------- recycling (A8)

def test_recycle_generator_matches_published_vector(po):
    vec = [int(l, 16) for l in open(os.path.join(GOLD, "splitmix64.txt")) if l.strip() and not l.startswith("#")]
    gam = 0x9E3779B97F4A7C15
    got = [po.mix64((k * gam) & 0xFFFFFFFFFFFFFFFF) for k in range(3)]
    assert got == vec
    u = np.array([po.recycle_uniform(3004, i, 7, j) for i in range(2000) for j in range(3)])
    assert 0.0 <= u.min() and u.max() < 1.0
    assert abs(u.mean() - 0.5) < 0.02 and abs(u.var() - 1 / 12) < 0.005


def test_outflow_recycling(po):
    """particles leaving through the outflow face re-enter in a random cell of the inflow
    boundary with inflow conditions; N constant; id kept."""
    n = [16, 8]; h = 1.0 / 8
    cfg = _cfg(2, n, h, [[2, 3], [1, 1]], inflow_rho=1.4, inflow_p=1.0, inflow_v=[3.0, 0.0, 0.0],
               recycle_seed=3004, ppc_inflow=4.0)
    o = po.Oracle(cfg)
    rng = np.random.default_rng(4)
    N = 16 * 8 * 4
    x = rng.uniform(0, 1, (2, N)) * np.array([[2.0], [1.0]])
    v = np.zeros((2, N)); v[0] = 3.0
    rho = np.full(N, 1.4); mass = rho * h * h / 4; e = np.full(N, 1.0 / (0.4 * 1.4))
    o.load_particles(x, v, mass, rho, e)
    o.step(0.0, 0.3, 40)
    s = o.stats()
    assert s.n_recycled > 50
    X = o.particles(po.P_X)
    assert X.shape[1] == N and (X[0] >= 0).all() and (X[0] <= 2.0).all() and (X[1] >= 0).all() and (X[1] <= 1.0).all()
    # one more step, watch who gets recycled
    x_before = X.copy()
    o.step(0.0, 0.3, 1)
    X2 = o.particles(po.P_X)
    rec = (X2[0] < x_before[0] - 1.0)
    assert rec.any()
    assert (X2[0][rec] <= h).all()
    np.testing.assert_array_equal(o.particles(po.P_RHO)[rec], 1.4)
    np.testing.assert_array_equal(o.particles(po.P_V)[0][rec], 3.0)
    np.testing.assert_array_equal(o.particles(po.P_Q)[rec], 0.0)
    np.testing.assert_allclose(o.particles(po.P_M)[rec], 1.4 * h * h / 4.0, rtol=1e-15)


# --------------------------------------------------------------------------- derived normals (A7)

def test_derived_normals_point_outward(po):
    """Normals derived from a disc mask: unit length, within 25 degrees of the radial direction on average
    at the nodes that touch both masked and unmasked cells, pointing OUT of the obstacle."""
    n = [48, 48]; h = 1.0 / 48
    ii = np.arange(48) + 0.5
    mask = ((ii[None, :] - 24) ** 2 + (ii[:, None] - 24) ** 2 <= 10 ** 2).astype(np.uint8)
    o = po.Oracle(_cfg(2, n, h, [[3, 3], [3, 3]], obstacle_mask=mask))
    nrm = o.grid(po.G_NORMAL).reshape(2, 49, 49)
    flag = o.grid(po.G_FLAG).reshape(49, 49) > 0
    g = np.arange(49) - 24.0
    R = np.sqrt(g[None, :] ** 2 + g[:, None] ** 2)
    surf = flag & (R > 9.0)
    rad = np.stack([np.broadcast_to(g[None, :], R.shape), np.broadcast_to(g[:, None], R.shape)]) / np.where(R > 0, R, 1)
    ln = np.sqrt((nrm ** 2).sum(axis=0))
    np.testing.assert_allclose(ln[surf], 1.0, rtol=1e-12)
    cosang = (nrm * rad).sum(axis=0)[surf]
    assert cosang.min() > 0.5 and np.degrees(np.arccos(np.clip(cosang, -1, 1))).mean() < 25.0


# --------------------------------------------------------------------------- Sod tube vs the exact Riemann solution

def test_riemann_solver_against_published_star_state():
    gold = {}
    for line in open(os.path.join(GOLD, "sod_exact_star.txt")):
        if line.strip() and not line.startswith("#"):
            k, v, tol = line.split()
            gold[k] = (float(v), float(tol))
    ps, us, rl, rr = riemann.star_state(1.0, 0.0, 1.0, 0.125, 0.0, 0.1, 1.4)
    shock, head, tail = riemann.sod_wave_speeds(1.4)
    got = dict(p_star=ps, u_star=us, rho_starL=rl, rho_starR=rr, shock_speed=shock,
               rarefaction_head=head, rarefaction_tail=tail)
    for k, (v, tol) in gold.items():
        assert abs(got[k] - v) <= tol, (k, got[k], v)


def _run_sod_to(po, nx, ny, tf, jitter=0.0, jitter_y=True, cfl=0.3):
    w = inputs.sod(nx=nx, ny=ny, jitter=jitter, jitter_y=jitter_y)
    o = po.Oracle(w["cfg"])
    o.load_particles(w["x"], w["v"], w["mass"], w["rho"], w["e"])
    h = w["cfg"]["dx"]
    while True:
        s = o.stats()
        dtn = cfl * h / (s.vmax + s.cmax)
        if s.t + dtn >= tf:
            o.step(tf - s.t, cfl, 1)
            break
        o.step(0.0, cfl, 1)
    return o, w


def _sod_l1(po, o, t):
    rho = o.particles(po.P_RHO); x = o.particles(po.P_X); m = o.particles(po.P_M)
    vol = m / rho
    ex, _, _ = riemann.sample((x[0] - 0.5) / t, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1)
    return (vol * np.abs(rho - ex)).sum() / vol.sum()


def test_sod_against_exact_solution_paper_setup(po):
    """The paper's own Sod run: 1 x 100 cells, regular particle lattice, t = 0.143, compared with the
    exact solution.  Bound B = 1.25 x the value the oracle gave when it was frozen (0.02868);
    the L1 error falls under refinement 25 -> 50 cells (0.0398 -> 0.0284) and has levelled off by 100.  Also pins the wave structure: plateau pressure
    and velocity near (p*, u*) and the shock position near 0.5 + S t.
    (Beyond ~100 cells the Q1 + FLIP scheme's cell-crossing noise makes the particle density error GROW with
    refinement -- a property of the method as published, recorded in DESIGN.md, not a defect to pin.)"""
    errs = []
    for nx in (25, 50, 100):
        o, w = _run_sod_to(po, nx, 1, 0.143)
        errs.append(_sod_l1(po, o, 0.143))
    assert errs[0] > 1.3 * errs[1] and errs[2] < 1.05 * errs[1], errs
    assert errs[2] <= 1.25 * 0.02868, errs
    x = o.particles(po.P_X)[0]; v = o.particles(po.P_V)[0]
    rho = o.particles(po.P_RHO); e = o.particles(po.P_E)
    ps, us, _, _ = riemann.star_state(1.0, 0.0, 1.0, 0.125, 0.0, 0.1)
    shock, head, tail = riemann.sod_wave_speeds()
    # Star region either side of the contact.  The particle variable rho is a passive diagnostic in this scheme
    # (the force uses (P+Q) M / rho = ((gamma-1) E + Q/rho) M), so the wave structure is pinned through
    # u and the specific internal energy E, whose exact star values are p*/((gamma-1) rho*_{L,R}).
    _, _, rsl, rsr = riemann.star_state(1.0, 0.0, 1.0, 0.125, 0.0, 0.1)
    xc = 0.5 + us * 0.143
    left = (x > 0.5 + (tail + 0.1) * 0.143) & (x < xc - 0.02)
    right = (x > xc + 0.02) & (x < 0.5 + (shock - 0.2) * 0.143)
    assert left.sum() >= 8 and right.sum() >= 8
    assert abs(v[left].mean() - us) < 0.08 * us and abs(v[right].mean() - us) < 0.08 * us
    assert abs(e[left].mean() - ps / (0.4 * rsl)) < 0.06 * ps / (0.4 * rsl)
    assert abs(e[right].mean() - ps / (0.4 * rsr)) < 0.06 * ps / (0.4 * rsr)
    # undisturbed states outside the wave fan
    assert np.abs(rho[x < 0.5 + (head - 0.25) * 0.143] - 1.0).max() < 1e-3
    assert np.abs(rho[x > 0.5 + (shock + 0.6) * 0.143] - 0.125).max() < 0.02   # Landshoff precursor (c1 = 1)
    # shock position: where u falls through u*/2
    xs = np.sort(x[(v > 0.4 * us) & (x > 0.6)])
    assert abs(xs[-1] - (0.5 + shock * 0.143)) < 0.06   # shock smeared over ~5 cells of h = 0.01


def test_sod_grid_density_falls_under_refinement(po):
    """north_star: 'L1 density error within a stated bound that falls under refinement'.  The quantity Fig. 5 plots is
    the density 'interpolated on the grid' (reading A18); the one the method itself controls is the
    nodal mass density m_i / h^d after a P2G at the final positions (eq. 14): on the paper's set-up
    (1 row of cells, regular lattice, t = 0.143) its L1 distance to the exact solution falls strictly
    from 25 to 200 cells with an observed order >= 0.5 between 25 and 100 cells.  (The PARTICLE density of
    test_sod_against_exact_solution_paper_setup does not: see DESIGN.md 2.2.)  Bound at 100 cells: 1.25 x 0.0188."""
    errs = []
    for nx in (25, 50, 100, 200):
        o, w = _run_sod_to(po, nx, 1, 0.143)
        h = w["cfg"]["dx"]
        o.grid_reset(); o.p2g1()
        rho_g = o.grid(po.G_MASS).reshape(o.nn[1], o.nn[0])[0] / h ** 2      # y periodic with one row: dual cell h x h
        xi = np.arange(o.nn[0]) * h
        ex, _, _ = riemann.sample((xi - 0.5) / 0.143, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1)
        errs.append(np.abs(rho_g - ex)[1:-1].sum() * h)                      # wall nodes have half a dual cell: left out
    assert errs[0] > errs[1] > errs[2] > errs[3], errs
    assert np.log2(errs[0] / errs[2]) / 2.0 >= 0.5, errs
    assert errs[2] <= 1.25 * 0.0188, errs


def test_sod_config1_jittered_bound(po):
    """BASELINE config 1 itself (256 x 4, jitter 0.1 dx, CFL 0.3, 100 steps): L1 density error vs the exact solution
    at the reached time stays under B = 1.25 x the frozen oracle value (0.1091)."""
    w = inputs.sod()
    o = po.Oracle(w["cfg"])
    o.load_particles(w["x"], w["v"], w["mass"], w["rho"], w["e"])
    o.step(0.0, w["cfl"], 100)
    s = o.stats()
    err = _sod_l1(po, o, s.t)
    assert err <= 1.25 * 0.1091, err
    assert s.n_negjac == 0 and s.n_nonfinite == 0
