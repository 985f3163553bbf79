"""CUDA-vs-oracle parity of the Yee field update (pic_update_fields) and of the
self-consistent loop (option field_update), through the C ABI.

Tolerance of the fields: one update rounds E + dt*(curl B - J) and twice B - dt/2*curl E
in fp32 — a handful of half-ulp errors of max|F| each — and the scheme does not amplify them, so after n
updates |F_gpu - F_oracle| <= n * 1e-6 * max(|E|, |B|, dt*|J|) (measured: ~1.5e-7 per update).
"""
import math

import numpy as np
import pytest
import torch

import oracle
import pic_parity as PP
from oracle import yee_oracle as Y
from paper_2110_08650_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL_F = 1e-6


def _vacuum(grid, order):
    from paper_2110_08650_b200.binding import Pic
    wl = W.CONFIGS["thermal_128"].scaled(grid, shape_order=order)
    return wl, Pic(wl.grid, wl.cell, wl.dt, wl.supercell, wl.shape_order, max_particles=0)


@pytest.mark.parametrize("grid", [(16, 16, 8), (40, 24, 20), (64, 16, 12), (8, 8, 4), (72, 40, 80)])
@pytest.mark.parametrize("order,tile", ((2, 8), (3, 8), (2, 16), (3, 16)))
def test_vacuum_update_matches_oracle(grid, order, tile):
    """No particles (J = 0): grids smaller than one 32 x tile tile, ragged tiles, several tiles, several z chunks."""
    wl, pic = _vacuum(grid, order)
    pic.set_option("yee_tile", tile)
    F0 = W.make_fields(wl)
    pic.set_fields(F0.cuda().contiguous())
    F = [f.astype(np.float64) for f in F0.numpy()]
    zero = [np.zeros_like(F[0])] * 3
    scale = max(np.abs(f).max() for f in F)
    for n in range(1, 6):
        pic.update_fields()
        F = Y.yee_update(F, zero, wl.dt, wl.cell)
        G = pic.get_fields().cpu().numpy().astype(np.float64)
        err = np.abs(G - np.stack(F)).max()
        assert err <= n * TOL_F * scale, (n, err / scale)
    pic.sync()
    pic.destroy()


@pytest.mark.parametrize("grid", [(64, 16, 12), (72, 40, 80), (136, 24, 8), (40, 24, 20)])
@pytest.mark.parametrize("order,tile,wide", ((2, 8, 1), (3, 8, 1), (2, 16, 1), (3, 16, 1), (2, 8, 0), (3, 16, 0)))
def test_update_with_a_given_current_matches_oracle(grid, order, tile, wide):
    """A random J set through set_current before every update: the J term and its indexing (unpadded, off the padded
    arrays' 16-byte grid by pad_lo_x) in both field kernels — one cell per thread, and four per thread on grids at
    least 64 wide (one tile, ragged second tile, two tiles and a rest; the last grid is too narrow and falls back)."""
    wl, pic = _vacuum(grid, order)
    pic.set_option("yee_tile", tile)
    pic.set_option("yee_wide", wide)
    F0 = W.make_fields(wl)
    pic.set_fields(F0.cuda().contiguous())
    F = [f.astype(np.float64) for f in F0.numpy()]
    scale = max(np.abs(f).max() for f in F)
    nx, ny, nz = grid
    g = torch.Generator().manual_seed(nx * 7 + order)
    for n in range(1, 5):
        J = (torch.rand((3, nz, ny, nx), generator=g) - 0.5) * float(scale)
        pic.set_current(J.cuda().contiguous())
        pic.update_fields()
        F = Y.yee_update(F, [j.astype(np.float64) for j in J.numpy()], wl.dt, wl.cell)
        G = pic.get_fields().cpu().numpy().astype(np.float64)
        err = np.abs(G - np.stack(F)).max()
        assert err <= n * TOL_F * scale, (n, err / scale)
    pic.sync()
    pic.destroy()


def test_index64_variant_matches_the_default_bit_for_bit():
    """The 64-bit-index instantiation (taken by itself beyond 2^32 elements) on a small grid and on one the
    four-cell kernel takes."""
    for grid in ((40, 24, 20), (72, 24, 20)):
        out = []
        for idx64 in (0, 1):
            wl, pic = _vacuum(grid, 3)
            pic.set_option("yee_index64", idx64)
            pic.set_fields(W.make_fields(wl).cuda().contiguous())
            for _ in range(3):
                pic.update_fields()
            out.append(pic.get_fields().cpu())
            pic.destroy()
        assert torch.equal(out[0], out[1])


@pytest.mark.parametrize("name", ("lwfa", "pqs_large"))
def test_full_size_grid_sampled_boxes(name):
    """The grids of configs[2] and configs[4] (67 M cells, the launch configuration bench.py times: 64-plane z chunks),
    two updates of seeded random fields (no particles: J = 0) against the oracle on sampled boxes: the update of a cell depends on cells within 2 of it per update, so the oracle run on a
    box cut out of the global arrays (wrapped periodically) is exact 4 cells inside the box."""
    from paper_2110_08650_b200.binding import Pic
    wl = W.CONFIGS[name]
    nx, ny, nz = wl.grid
    pic = Pic(wl.grid, wl.cell, wl.dt, wl.supercell, wl.shape_order, max_particles=0)
    g = torch.Generator(device="cuda").manual_seed(5)
    F0 = (torch.rand((6, nz, ny, nx), device="cuda", generator=g) - 0.5) * 0.1
    pic.set_fields(F0)
    n_up, B, M = 2, 24, 4
    for _ in range(n_up):
        pic.update_fields()
    G = pic.get_fields()
    pic.sync()
    # boxes at the periodic corner, across the z-chunk boundary at k = 64, and in the interior
    for lo in ((-12, -12, -12), (100, 500, 52), (nx - 20, 7, nz - 10), (31, ny - 13, 120)):
        ix = torch.arange(lo[0], lo[0] + B, device="cuda") % nx
        iy = torch.arange(lo[1], lo[1] + B, device="cuda") % ny
        iz = torch.arange(lo[2], lo[2] + B, device="cuda") % nz
        cut = lambda A: A[:, iz][:, :, iy][:, :, :, ix].cpu().numpy().astype(np.float64)
        F = list(cut(F0))
        zero = [np.zeros_like(F[0])] * 3
        for _ in range(n_up):
            F = Y.yee_update(F, zero, wl.dt, wl.cell)
        got = cut(G)[:, M:-M, M:-M, M:-M]
        exp = np.stack(F)[:, M:-M, M:-M, M:-M]
        err = np.abs(got - exp).max() / 0.05
        assert err <= n_up * TOL_F, (lo, err)
    pic.destroy()


def test_plane_wave_against_the_closed_form():
    """40 updates of a discrete plane wave (oblique k) against the analytic solution with the numerical
    dispersion relation (derivation: tests/test_oracle_yee.py) — no oracle involved."""
    from test_oracle_yee import _plane_wave
    grid = (32, 16, 8)
    wl, pic = _vacuum(grid, 2)
    at, w = _plane_wave(grid, wl.cell, wl.dt, (2, -1, 1), pol_seed=3)
    F0 = np.stack(at(0))
    scale = np.abs(F0).max()
    pic.set_fields(torch.from_numpy(F0.astype(np.float32)).cuda().contiguous())
    for n in range(1, 41):
        pic.update_fields()
    G = pic.get_fields().cpu().numpy().astype(np.float64)
    err = np.abs(G - np.stack(at(40))).max()
    print(f"\n[plane wave, 40 updates] err/max|F| = {err / scale:.3e}")
    # the initial state itself is rounded to fp32 (6e-8 relative), then 40 updates
    assert err <= 41 * TOL_F * scale
    pic.destroy()


def _loop_case(order, grid=(24, 16, 12), ppc=8, weight=0.01):
    wl = W.CONFIGS["thermal_128"].scaled(grid, shape_order=order, ppc=ppc)
    parts, fields = W.make_particles(wl), W.make_fields(wl)
    parts.w.mul_(weight)       # omega_p*dt = sqrt(ppc*w)*dt = 0.14: a stable, weakly coupled plasma
    return wl, parts, fields


@pytest.mark.parametrize("order", (1, 2, 3))
@pytest.mark.parametrize("mode", ("option_tma", "option_plain_loads", "explicit_calls"))
def test_self_consistent_loop(order, mode):
    """Ten steps of push + deposit + field update on both sides, free-running."""
    n_steps = 10
    wl, parts, fields = _loop_case(order)
    orc = PP.oracle_for(wl, parts, fields)
    opts = {"tma": 0} if mode == "option_plain_loads" else {}
    pic = PP.gpu_for(wl, parts, fields, **opts)
    assert orc.step(n_steps, update_fields=True) == 0
    if mode == "explicit_calls":
        for _ in range(n_steps):
            pic.step(1)
            pic.update_fields()
    else:
        pic.set_option("field_update", 1)
        pic.step(n_steps)
    pic.sync()
    rep = PP.compare(wl, orc, pic, n_steps, 0.05)
    G = pic.get_fields().cpu().numpy().astype(np.float64)
    Fo = np.stack(orc.fields)
    scale = np.abs(Fo).max()
    f_err = np.abs(G - Fo).max() / scale
    print(f"\n[loop order={order} {mode}] {rep}  fields err/max|F|={f_err:.3e}")
    assert rep.max_dx <= n_steps * PP.TOL_X and rep.max_du_rel <= n_steps * PP.TOL_U
    assert rep.j_err_rel <= PP.TOL_J10
    assert rep.n_member_mismatch == 0 and rep.counts_equal_outside_band
    assert f_err <= n_steps * TOL_F
    # the fields did change: this is not the static-field path
    assert np.abs(Fo - fields.numpy()).max() > 0.05 * scale
    pic.destroy()


@pytest.mark.parametrize("order", (2, 3))
def test_gauss_law_is_kept_on_the_gpu(order):
    """div E - rho at the nodes stays what it was: the GPU's Esirkepov J and its field update use the same
    discrete divergence.  rho in fp64 from the GPU's own positions (S22's recipe)."""
    wl, parts, fields = _loop_case(order)
    pic = PP.gpu_for(wl, parts, fields, field_update=1)
    prm = oracle.OracleParams.make(wl.grid, wl.cell, wl.dt, wl.supercell, wl.shape_order)

    def gauss():
        P = PP.gpu_particles_by_id(pic)
        rho = oracle.rho(prm, P["x"], P["y"], P["z"], -P["w"].astype(np.float64))
        E = pic.get_fields().cpu().numpy().astype(np.float64)[:3]
        return Y.div_E(*E, wl.cell) - rho, np.abs(rho).max()

    g0, rmax = gauss()
    n_steps = 5
    pic.step(n_steps)
    pic.sync()
    g1, _ = gauss()
    drift = np.abs(g1 - g0).max() / rmax
    print(f"\n[gauss order={order}] drift of (div E - rho) / max|rho| after {n_steps} steps = {drift:.3e}")
    assert drift <= n_steps * PP.TOL_CONT
    pic.destroy()


def test_energies_after_forty_self_consistent_steps():
    """Free-running 40 steps of the warm dilute plasma (tests/pic_parity.py): electric, magnetic and kinetic energy
    of the GPU state against the oracle's, each to 1e-5 relative (integrated quantities: the per-particle and
    per-cell rounding differences average out), and the total within 1 % of its initial value."""
    wl, parts, fields = PP.warm_dilute_plasma(2)
    orc = PP.oracle_for(wl, parts, fields)
    pic = PP.gpu_for(wl, parts, fields, field_update=1)
    e_start = PP.energies(fields.numpy(), parts.ux.numpy(), parts.uy.numpy(), parts.uz.numpy(), parts.w.numpy(), wl.cell)
    assert orc.step(40, update_fields=True) == 0
    pic.step(40)
    pic.sync()
    G = PP.gpu_particles_by_id(pic)
    eg = PP.energies(pic.get_fields().cpu().numpy(), G["ux"], G["uy"], G["uz"], G["w"], wl.cell)
    O = orc.particles()
    eo = PP.energies(orc.fields, O["ux"], O["uy"], O["uz"], O["w"], wl.cell)
    print(f"\n[energies after 40 steps] gpu {eg}  oracle {eo}  start {e_start}")
    for a, b in zip(eg, eo):
        assert abs(a - b) <= 1e-5 * abs(b)
    assert abs(sum(eg) / sum(e_start) - 1) < 1e-2
    pic.destroy()


def test_full_size_self_consistent_loop_keeps_gauss_law():
    """configs[1] at full size (128^3 cells, 33.5 M particles, TSC; weights scaled to omega_p*dt = 0.2 so that the closed
    loop is stable), three steps with option field_update in the launch configuration bench.py --self-consistent times.
    Properties that hold at any size: no device fault, ids a permutation, membership consistent; and on a sampled box
    div E - rho (rho in fp64 from the GPU's own positions, all particles within reach of the box) stays what it was."""
    from paper_2110_08650_b200.binding import Pic
    wl = W.CONFIGS["thermal_128"]
    n = W.n_particles(wl)
    dev = "cuda:0"
    pic = Pic(wl.grid, wl.cell, wl.dt, wl.supercell, wl.shape_order, max_particles=n, device=dev)
    keys = ("x", "y", "z", "ux", "uy", "uz", "w", "species")
    for chunk in W.particle_chunks(wl, device=dev, max_chunk=1 << 23):
        chunk.w.mul_(0.01)
        pic.load_particles(*(getattr(chunk, k) for k in keys))
        pic.sync()
    del chunk
    pic.set_fields(W.make_fields(wl, device=dev))
    pic.set_option("field_update", 1)
    lo, B, M = (50, 60, 28), 24, 4          # box spans supercell faces and the z-chunk boundary of the Yee kernel at k = 32
    prm = oracle.OracleParams.make((B, B, B), wl.cell, wl.dt, wl.supercell, wl.shape_order)

    def gauss():
        P = pic.get_particles()
        inb = torch.ones(P["x"].numel(), dtype=torch.bool, device=dev)
        for a, k in enumerate("xyz"):
            inb &= (P[k] >= lo[a]) & (P[k] < lo[a] + B)
        q = {k: P[k][inb].cpu().numpy() for k in ("x", "y", "z", "w")}
        rho = oracle.rho(prm, q["x"] - lo[0], q["y"] - lo[1], q["z"] - lo[2], -q["w"].astype(np.float64))
        E = pic.get_fields()[:3, lo[2] - 1:lo[2] + B, lo[1] - 1:lo[1] + B, lo[0] - 1:lo[0] + B].cpu().numpy().astype(np.float64)
        div = ((E[0][1:, 1:, 1:] - E[0][1:, 1:, :-1]) + (E[1][1:, 1:, 1:] - E[1][1:, :-1, 1:])
               + (E[2][1:, 1:, 1:] - E[2][:-1, 1:, 1:]))
        sl = (slice(M, -M),) * 3
        return (div - rho)[sl], float(np.abs(rho[sl]).max())

    g0, rmax = gauss()
    n_steps = 3
    pic.step(n_steps)
    pic.sync()
    st = pic.get_stats()
    assert st["error"] == 0 and st["particles"] == n and st["steps"] == n_steps
    g1, _ = gauss()
    drift = float(np.abs(g1 - g0).max()) / rmax
    print(f"\n[full-size loop] drift of (div E - rho) / max|rho| in the box after {n_steps} steps = {drift:.3e}")
    assert drift <= n_steps * PP.TOL_CONT
    ids = pic.get_particles()["id"].to(torch.int64) & 0xFFFFFFFF
    assert torch.equal(torch.sort(ids).values, torch.arange(n, device=dev))
    assert PP.gpu_membership_consistent(wl, pic)
    pic.destroy()


def test_update_before_set_fields_is_a_state_error():
    from paper_2110_08650_b200.binding import Pic, PicError
    pic = Pic((16, 16, 8), shape_order=1, max_particles=0)
    with pytest.raises(PicError):
        pic.update_fields()
    with pytest.raises(PicError):
        pic.get_fields()
    with pytest.raises(PicError):
        pic.set_option("yee_tile", 5)
    pic.destroy()
