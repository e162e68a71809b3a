"""Longer validation workloads, on the oracle and through the CUDA path.

* Sod shock tube as the paper runs it -- 1 x 100 cells, regular particle lattice, t = 0.143 -- for the
  four artificial-viscosity settings of Fig. 9, (c0, c1) = (1,1), (0,0), (10,0), (0,10): the qualitative
  ordering of the figure on the oracle (CPU), and GPU-vs-oracle parity at t = 0.143 for each setting (GPU).
* Sedov blast at 64^3 run until the shock has crossed 0.3 of the box: the similarity law R(t) ~ (E t^2 / rho)^(1/5)
  (GPU; the constant is fitted from the run, not quoted).

Reading recorded in DESIGN.md: with eq. (4) as printed and c1 = 10 the explicit linear viscosity violates its own diffusive
stability limit dt <= h / (2 c1 c_s) at the paper's CFL numbers (at alpha = 0.3 the oracle's energies grow by 40 orders of
magnitude in 100 steps and time stands still near t = 0.008),
so the (0,10) case runs at alpha = 0.02 on both sides; the other three use alpha = 0.3.  (At alpha = 0.04 that case
reaches t = 0.143 but sits on the stability margin: a 1e-14 perturbation of the input grows to 1e-4 by the end, which makes
any two correct implementations disagree; at alpha = 0.02 the same perturbation stays at 5e-15.)
"""
import numpy as np
import pytest

import riemann
from paper_2404_17057_b200 import inputs

T_END = 0.143
CASES = {(1.0, 1.0): 0.3, (0.0, 0.0): 0.3, (10.0, 0.0): 0.3, (0.0, 10.0): 0.02}      # (c0, c1) -> alpha


def _sod_paper(c0, c1):
    w = inputs.sod(nx=100, ny=1, jitter=0.0)
    cfg = dict(w["cfg"], c0=c0, c1=c1)
    return w, cfg


def _run_to(solver, stats, tf, alpha, h):
    """CFL steps until the next one would pass tf, then one fixed step that lands on tf (both sides the same way)."""
    n = 0
    while True:
        s = stats()
        dtn = alpha * h / (s.vmax + s.cmax)
        n += 1
        if s.t + dtn >= tf:
            solver.step(tf - s.t, alpha, 1)
            return n
        solver.step(0.0, alpha, 1)


def _star_variation(x, u):
    """Total variation of the particle velocity between the tail of the rarefaction and the shock: 0 for the exact
    solution (u = u* there), large when the post-shock state rings."""
    shock, head, tail = riemann.sod_wave_speeds()
    idx = np.argsort(x)
    xs, us = x[idx], u[idx]
    star = (xs > 0.5 + (tail + 0.1) * T_END) & (xs < 0.5 + (shock - 0.15) * T_END)
    assert star.sum() > 60
    return np.abs(np.diff(us[star])).sum()


def test_sod_viscosity_sweep_ordering_on_the_oracle(po):
    """Fig. 9, qualitatively: without artificial viscosity the post-shock state oscillates most; either
    term damps the oscillations; the linear term with c1 = 10 smears the profile most (largest L1 density error)."""
    tv, l1 = {}, {}
    for (c0, c1), alpha in CASES.items():
        w, cfg = _sod_paper(c0, c1)
        o = po.Oracle(cfg)
        o.load_particles(w["x"], w["v"], w["mass"], w["rho"], w["e"])
        _run_to(o, o.stats, T_END, alpha, cfg["dx"])
        s = o.stats()
        assert abs(s.t - T_END) < 1e-12 and s.n_nonfinite == 0 and s.n_negjac == 0
        x, u, rho, m = o.particles(po.P_X)[0], o.particles(po.P_V)[0], o.particles(po.P_RHO), o.particles(po.P_M)
        tv[(c0, c1)] = _star_variation(x, u)
        ex, _, _ = riemann.sample((x - 0.5) / T_END, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1)
        vol = m / rho
        l1[(c0, c1)] = (vol * np.abs(rho - ex)).sum() / vol.sum()
    assert tv[(0.0, 0.0)] > 1.3 * tv[(10.0, 0.0)] > 1.3 * tv[(1.0, 1.0)] > 1.3 * tv[(0.0, 10.0)], tv
    assert l1[(0.0, 10.0)] > 1.25 * max(l1[(1.0, 1.0)], l1[(0.0, 0.0)], l1[(10.0, 0.0)]), l1
    assert max(l1.values()) < 0.06, l1


def test_sod_linear_viscosity_c1_10_is_unstable_at_the_papers_cfl(po):
    """The reading recorded above: (c0, c1) = (0, 10) at alpha = 0.3 leaves the explicit stability region."""
    w, cfg = _sod_paper(0.0, 10.0)
    o = po.Oracle(cfg)
    o.load_particles(w["x"], w["v"], w["mass"], w["rho"], w["e"])
    o.step(0.0, 0.3, 120)
    s = o.stats()
    e = o.particles(po.P_E)
    # exponential growth of the specific energy at the shock; the CFL step collapses and time stands still near t = 0.008
    assert (not np.isfinite(e).all()) or (np.nanmax(e) > 1e20 and s.t < 0.01)


@pytest.mark.gpu
@pytest.mark.parametrize("c0,c1", list(CASES.keys()))
def test_sod_paper_setup_gpu_vs_oracle(po, mpm, c0, c1):
    """The paper's own Sod run through the CUDA path (TILED family) against the oracle at t = 0.143: 1e-9 relative L1 on
    rho, u, E by particle id, same number of steps, and the GPU result obeys the oracle's error bound against the exact solution."""
    alpha = CASES[(c0, c1)]
    w, cfg = _sod_paper(c0, c1)
    o = po.Oracle(cfg)
    o.load_particles(w["x"], w["v"], w["mass"], w["rho"], w["e"])
    g = mpm.Solver(cfg, sort_every=1, variant=mpm.VARIANT_TILED)
    g.load_particles(w["x"], w["v"], w["mass"], w["rho"], w["e"])
    no = _run_to(o, o.stats, T_END, alpha, cfg["dx"])
    # the GPU takes the same NUMBER of steps (the oracle's stopping decision t + dt >= T_END can fall either way when it
    # is within rounding), each with its own device-side CFL dt, and the same closing step onto T_END
    g.step(0.0, alpha, no - 1)
    sg = g.stats()
    assert T_END - sg.t > 0.0 and T_END - sg.t <= 1.0001 * sg.dt_next
    g.step(T_END - sg.t, alpha, 1)
    so, sg = o.stats(), g.stats()
    assert so.step == sg.step and abs(so.t - sg.t) <= 1e-12 and sg.n_nonfinite == 0 and sg.n_out_of_cell == 0
    p = g.read_particles()
    for key, fo in (("rho", po.P_RHO), ("e", po.P_E), ("v", po.P_V), ("x", po.P_X)):
        a = o.particles(fo)
        assert np.abs(a - p[key]).sum() <= 1e-9 * np.abs(a).sum(), (c0, c1, key, np.abs(a - p[key]).sum() / np.abs(a).sum())
    ex, _, _ = riemann.sample((p["x"][0] - 0.5) / T_END, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1)
    vol = p["mass"] / p["rho"]
    assert (vol * np.abs(p["rho"] - ex)).sum() / vol.sum() < 0.06


@pytest.mark.gpu
def test_sedov_similarity_law(mpm):
    """3D point blast in a cold gas (config 4's recipe at 64^3, ambient p = 1e-5, E = 1, rho = 1): the shock radius follows
    R(t) = xi0 (E t^2 / rho)^(1/5).  R = radius of the density maximum of the radially binned particle density (parabolic
    peak fit), sampled every 100 steps from step 200 (R ~ 0.13) until R > 0.33.  Asserted: the log-log slope of R(t) is
    2/5 within 0.02, and xi = R / (E t^2 / rho)^(1/5) stays within 4 % of its mean (the constant is fitted, not quoted;
    the scheme loses ~8 % of the total energy over the run, 1.6 % in R)."""
    n = 64
    w = inputs.sedov(n=n)
    h = w["cfg"]["dx"]
    g = mpm.Solver(w["cfg"], sort_every=1, variant=mpm.VARIANT_TILED)
    g.load_particles(w["x"], w["v"], w["mass"], w["rho"], w["e"])
    g.step(0.0, w["cfl"], 100)
    ts, Rs = [], []
    for it in range(20):
        g.step(0.0, w["cfl"], 100)
        st = g.stats()
        assert st.n_nonfinite == 0 and st.n_negjac == 0 and st.n_out_of_cell == 0
        p = g.read_particles(mpm.P_X | mpm.P_RHO)
        r = np.sqrt(((p["x"] - 0.5) ** 2).sum(axis=0))
        b = np.minimum((r / h).astype(np.int64), n - 1)
        cnt = np.bincount(b, minlength=n)
        rho_b = np.bincount(b, weights=p["rho"], minlength=n) / np.maximum(cnt, 1)
        i = int(np.argmax(rho_b[: n // 2]))
        y0, y1, y2 = rho_b[i - 1], rho_b[i], rho_b[i + 1]
        shift = 0.5 * (y0 - y2) / (y0 - 2.0 * y1 + y2)
        ts.append(st.t)
        Rs.append((i + 0.5 + shift) * h)
        if Rs[-1] > 0.33:
            break
    ts, Rs = np.array(ts), np.array(Rs)
    assert len(ts) >= 8 and Rs[0] < 0.16 and Rs[-1] > 0.33
    slope = np.polyfit(np.log(ts), np.log(Rs), 1)[0]
    assert abs(slope - 0.4) < 0.02, slope
    xi = Rs / ts ** 0.4                   # E = rho = 1
    assert np.abs(xi / xi.mean() - 1.0).max() < 0.04, xi
    assert 0.9 < xi.mean() < 1.1, xi.mean()
