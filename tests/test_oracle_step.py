"""Whole-step pins of the oracle (SURVEY.md §8(c) steps 3-7 chained) and of the input
generators (shapes / counts / exact representability; no method arithmetic in them)."""
import math

import numpy as np
import pytest
import torch

import oracle
from paper_2110_08650_b200 import workloads as W


def _tiny(order=1, grid=(16, 16, 16), ppc=2, u_th=0.05, fields="modes"):
    return W.CONFIGS["tiny_thermal"].scaled(grid, shape_order=order, ppc=ppc, u_th=u_th, fields=fields,
                                            amplitude=0.05, n_modes=4)


def _oracle_for(wl, parts, fields):
    orc = oracle.Oracle(wl.grid, wl.cell, wl.dt, wl.supercell, wl.shape_order)
    orc.load_particles(*(getattr(parts, k).numpy() for k in ("x", "y", "z", "ux", "uy", "uz", "w")),
                       species=parts.species.numpy())
    orc.set_fields(fields.numpy())
    return orc


@pytest.mark.parametrize("order", (1, 2, 3))
def test_step_invariants(order):
    wl = _tiny(order)
    parts, fields = W.make_particles(wl), W.make_fields(wl)
    orc = _oracle_for(wl, parts, fields)
    n0 = orc.n
    x0 = [orc.particles()[k].copy() for k in "xyz"]
    qw = orc.q[orc.species] * orc._parts[6]
    rho0 = oracle.rho(orc.prm, *x0, qw)
    assert orc.step(1) == 0
    P = orc.particles()
    assert P["x"].size == n0
    for k, n in zip("xyz", wl.grid):
        assert (P[k] >= 0).all() and (P[k] < n).all()
    # membership == floor(X) div SC recomputed from the returned positions
    sc = wl.supercell
    nsx, nsy = wl.grid[0] // sc[0], wl.grid[1] // sc[1]
    exp = (np.floor(P["x"]).astype(int) // sc[0]) + nsx * ((np.floor(P["y"]).astype(int) // sc[1])
                                                            + nsy * (np.floor(P["z"]).astype(int) // sc[2]))
    assert np.array_equal(exp, P["supercell"])
    assert orc.counts().sum() == n0
    # whole-step continuity (periodic wrap included)
    rho1 = oracle.rho(orc.prm, P["x"], P["y"], P["z"], qw)
    Jx, Jy, Jz = orc.J
    div = (Jx - np.roll(Jx, 1, 2)) + (Jy - np.roll(Jy, 1, 1)) + (Jz - np.roll(Jz, 1, 0))
    drho = (rho1 - rho0) / wl.dt
    assert np.abs(drho + div).max() / np.abs(drho).max() < 1e-12


def test_step_uniform_fields_matches_single_particle_closed_path():
    """Config-1 fields: every particle sees exactly E=(0.01,0,0), B=(0,0,0.1) whatever its
    position, so the chained step must equal boris()+move() applied directly."""
    wl = W.CONFIGS["tiny_thermal"].scaled((16, 16, 16), ppc=1)
    parts, fields = W.make_particles(wl), W.make_fields(wl)
    orc = _oracle_for(wl, parts, fields)
    u0 = np.stack([parts.ux.numpy(), parts.uy.numpy(), parts.uz.numpy()], 1).astype(np.float64)
    X0 = np.stack([parts.x.numpy(), parts.y.numpy(), parts.z.numpy()], 1)
    orc.step(1)
    P = orc.particles()
    for p in (0, 17, 4095):
        # the field arrays are float32: the oracle sees float64(float32(0.01)) etc.
        E, B = (float(np.float32(0.01)), 0, 0), (0, 0, float(np.float32(0.1)))
        un = oracle.boris(u0[p], E, B, -1.0, 0.5)
        np.testing.assert_allclose((P["ux"][p], P["uy"][p], P["uz"][p]), un, rtol=0, atol=2e-17)
        X1 = X0[p] + un / math.sqrt(1 + un @ un) * 0.5
        np.testing.assert_allclose((P["x"][p], P["y"][p], P["z"][p]), np.mod(X1, 16.0), rtol=0, atol=1e-14)


def test_J_is_last_step_only():
    wl = _tiny(2)
    parts, fields = W.make_particles(wl), W.make_fields(wl)
    a, b = _oracle_for(wl, parts, fields), _oracle_for(wl, parts, fields)
    a.step(3)
    b.step(2)
    b.step(1)
    for ja, jb in zip(a.J, b.J):
        assert np.array_equal(ja, jb)


def test_generators_shapes_and_exactness():
    wl = W.CONFIGS["tiny_thermal"]
    p = W.make_particles(wl)
    assert p.n == 16 ** 3 * 8 == W.n_particles(wl)
    assert p.x.dtype == torch.float64 and p.ux.dtype == torch.float32 and p.species.dtype == torch.int32
    # integer cell + fp32 fraction: the fraction survives a float32 round trip exactly
    for a in (p.x, p.y, p.z):
        fr = a - torch.floor(a)
        assert torch.equal(fr.to(torch.float32).to(torch.float64), fr)
        assert float(a.min()) >= 0.0 and float(a.max()) < 16.0
    cells = (torch.floor(p.x) + 16 * (torch.floor(p.y) + 16 * torch.floor(p.z))).to(torch.int64)
    assert torch.equal(torch.bincount(cells, minlength=4096), torch.full((4096,), 8))
    assert abs(float(p.ux.std()) - 0.01) < 5e-4
    f = W.make_fields(wl)
    assert f.shape == (6, 16, 16, 16) and float(f[0].min()) == np.float32(0.01) and float(f[5].max()) == np.float32(0.1)
    # deterministic
    assert torch.equal(W.make_particles(wl).ux, p.ux)


def test_generators_other_layouts():
    khi = W.CONFIGS["khi"].scaled((32, 16, 8))
    p = W.make_particles(khi)
    assert p.n == 32 * 16 * 8 * 9
    inner = (p.x >= 8) & (p.x < 24)
    assert torch.equal(p.species[inner], torch.zeros(int(inner.sum()), dtype=torch.int32))
    assert abs(float(p.uy[inner].mean()) - 0.2 / math.sqrt(0.96)) < 1e-3
    assert abs(float(p.uy[~inner].mean()) + 0.2 / math.sqrt(0.96)) < 1e-3
    hot = W.CONFIGS["khi_hotspot"].scaled((64, 64, 32))
    ph = W.make_particles(hot)
    assert ph.n == 64 * 64 * 32 * 9
    sc = (torch.floor(ph.x) // 8 + 8 * (torch.floor(ph.y) // 8 + 8 * (torch.floor(ph.z) // 4))).to(torch.int64)
    cnt = torch.bincount(sc, minlength=512)
    top = cnt.sort(descending=True).values[:5].sum()
    assert abs(int(top) - ph.n // 2) <= 1                      # 1% of 512 supercells = 5 hold 50%
    lw = W.CONFIGS["lwfa"].scaled((16, 64, 16), ramp_cells=8)
    pl = W.make_particles(lw)
    assert pl.n == 16 * 48 * 16 * 2 and float(pl.y.min()) >= 16.0
    assert float(pl.w.max()) == 1.0 and float(pl.w.min()) >= 0.0 and float(pl.ux.abs().max()) == 0.0
    fl = W.make_fields(lw)
    assert float(fl[0].abs().max()) > 1.0 and float(fl[1].abs().max()) == 0.0
    fm = W.make_fields(W.CONFIGS["thermal_128"].scaled((16, 16, 16)))
    assert float(fm.abs().max()) <= 0.01 + 1e-7 and float(fm.abs().max()) > 1e-3


def test_step_uses_charge_over_mass_per_species():
    """Pins the per-species q/m inside Oracle.step: two species (q, m) = (-1, 1) and
    (2, 3).  (a) B = 0, uniform E: u_new - u = (q/m) E dt exactly (SURVEY.md §8(c) step 4 pin (iii));
    (b) E = 0, uniform B: |u| is kept and u turns by exactly 2 atan(|q/m| |B| dt / (2 gamma)) in the sense
    of -q/m (pin (ii)); (c) the deposited current still carries the CHARGE q (not q/m): total current
    sum J_a V = sum_p q w dX_a dx_a / dt (step 6 pin (iii)).  A step that used q, m or q*m for the push, or
    q/m for the deposit, fails one of them."""
    grid, dt = (8, 8, 8), 0.5
    q, m = np.array([-1.0, 2.0]), np.array([1.0, 3.0])
    rng = np.random.default_rng(5)
    n = 64
    X = rng.uniform(0, 8, (3, n))
    u0 = rng.normal(0, 0.3, (3, n))
    w = rng.uniform(0.5, 1.5, n)
    sp = (np.arange(n) % 2).astype(np.int32)
    qm = (q / m)[sp]
    for order in (1, 2, 3):
        # (a) impulse
        orc = oracle.Oracle(grid, dt=dt, order=order)
        orc.set_species(q, m)
        orc.load_particles(*X, *u0, w, species=sp)
        F = np.zeros((6,) + grid[::-1])
        E = np.array([0.02, -0.01, 0.03])
        for a in range(3):
            F[a] = E[a]
        orc.set_fields(F)
        assert orc.step(1) == 0
        P = orc.particles()
        un = np.stack([P["ux"], P["uy"], P["uz"]])
        np.testing.assert_allclose(un - u0, qm[None, :] * E[:, None] * dt, rtol=0, atol=1e-15)
        # (c) total current carries q (times w), not q/m
        g = np.sqrt(1 + (un ** 2).sum(0))
        dX = un / g * dt
        for a in range(3):
            np.testing.assert_allclose(orc.J[a].sum(), ((q[sp] * w) * dX[a]).sum() / dt, rtol=1e-12)
        # (b) rotation
        orc = oracle.Oracle(grid, dt=dt, order=order)
        orc.set_species(q, m)
        orc.load_particles(*X, *u0, w, species=sp)
        F = np.zeros((6,) + grid[::-1])
        Bz = 0.4
        F[5] = Bz
        orc.set_fields(F)
        assert orc.step(1) == 0
        P = orc.particles()
        un = np.stack([P["ux"], P["uy"], P["uz"]])
        np.testing.assert_allclose((un ** 2).sum(0), (u0 ** 2).sum(0), rtol=1e-14)
        np.testing.assert_allclose(un[2], u0[2], rtol=0, atol=1e-16)
        gam = np.sqrt(1 + (u0 ** 2).sum(0))
        ang = np.arctan2(un[1], un[0]) - np.arctan2(u0[1], u0[0])
        ang = (ang + np.pi) % (2 * np.pi) - np.pi
        # du/dt = (q/m) u x B / gamma: for B along +z the perpendicular momentum turns by -(q/m)|B|dt/gamma
        np.testing.assert_allclose(ang, -np.sign(qm) * 2 * np.arctan(np.abs(qm) * Bz * dt / (2 * gam)), rtol=0, atol=1e-13)
