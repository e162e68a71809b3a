"""One step of Algorithm 1 is local: P2G#1 reaches one cell, V' of the neighbouring particles -- which P2G#2
scatters -- one more.  So the outputs inside a box of cells depend only on the particles within two cells of it.  This is what
lets the GPU tests compare BASELINE.json configs 4 and 5 at FULL size with the oracle on sampled sub-regions
(tests/test_gpu_parity.py::test_full_size_sampled_parity); here the method itself is checked with the oracle alone: the
oracle on box + 2 cells reproduces the oracle on all particles inside the box, bit for bit (the particle order is kept, so
even the summation order agrees) -- and with a halo of one cell it does not."""
import numpy as np
import pytest

from oracle import pyoracle as po
from paper_2404_17057_b200 import inputs


def _run(w, lo, halo, size=4):
    cfg, h = w["cfg"], w["cfg"]["dx"]
    d = cfg["dim"]
    n = np.array(cfg["n"][:d])
    per = [cfg["bc"][a][0] == 0 for a in range(d)]
    full = po.Oracle(cfg)
    full.load_particles(w["x"], w["v"], w["mass"], w["rho"], w["e"])
    full.step(0.0, w["cfl"], 1)
    dt = full.stats().dt_last
    cells = [np.clip(np.floor(w["x"][a] / h), 0, n[a] - 1).astype(np.int32) for a in range(d)]
    sel = np.ones(w["mass"].shape[0], bool)
    inner = sel.copy()
    for a in range(d):
        rel = cells[a] - (lo[a] - halo)
        if per[a]:
            rel %= int(n[a])
        sel &= (rel >= 0) & (rel < size + 2 * halo)
        inner &= (rel >= halo) & (rel < size + halo)
    idx = np.nonzero(sel)[0]
    inn = inner[idx]
    o = po.Oracle(cfg)
    o.load_particles(w["x"][:, idx], w["v"][:, idx], w["mass"][idx], w["rho"][idx], w["e"][idx])
    o.step(dt, 0.0, 1)
    worst = 0.0
    for f in (po.P_RHO, po.P_E, po.P_Q, po.P_X, po.P_V):
        worst = max(worst, float(np.abs(full.particles(f)[..., idx[inn]] - o.particles(f)[..., inn]).max()))
    nn = [int(n[a]) if per[a] else int(n[a]) + 1 for a in range(d)]
    axes = []
    for a in range(d):
        i = np.arange(lo[a], lo[a] + size + 1)
        axes.append(i % n[a] if per[a] else i[i < nn[a]])
    node = axes[0][:, None] + nn[0] * axes[1][None, :]
    if d == 3:
        node = node[:, :, None] + nn[0] * nn[1] * axes[2][None, None, :]
    node = node.ravel()
    for f in (po.G_MASS, po.G_MOM, po.G_FORCE, po.G_MOM2):
        a_, b_ = full.grid(f).reshape(-1, full.num_nodes)[..., node], o.grid(f).reshape(-1, o.num_nodes)[..., node]
        worst = max(worst, float(np.abs(a_ - b_).max()))
    return worst, int(inn.sum())


@pytest.mark.parametrize("case", ["sedov_centre", "sedov_corner", "clumps_wrap", "box2d"])
def test_subregion_oracle_equals_full_oracle(case):
    if case == "sedov_centre":
        w, lo = inputs.sedov(n=20), (8, 8, 8)
    elif case == "sedov_corner":
        w, lo = inputs.sedov(n=20), (0, 0, 0)
    elif case == "clumps_wrap":
        w, lo = inputs.clumps(n=20, num_particles=60_001), (18, 3, 9)        # the box crosses the periodic boundary
    else:
        w, lo = inputs.periodic_box(n=32), (29, 11)
    worst, count = _run(w, lo, halo=2)
    assert count > 0 and worst == 0.0
    if case in ("sedov_centre", "clumps_wrap", "box2d"):      # one cell of halo is not enough (the blast centre / moving gas)
        assert _run(w, lo, halo=1)[0] > 0.0
