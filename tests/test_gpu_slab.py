"""Slab decomposition on the GPU: two and four ranks EMULATED IN ONE PROCESS on one device (the
ranks step one after the other and exchange through slab.LoopbackExchange — nothing waits on anything, see
B200_PROFILING.md on emulating ranks), each rank stepping its slab + guards with the CUDA library.  The decomposed
run must reproduce the single-domain run of the same library: particles by global id, J plane by plane."""
import numpy as np
import pytest
import torch

import pic_parity as PP
from paper_2110_08650_b200 import slab as SL
from paper_2110_08650_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("world", (2, 4))
@pytest.mark.parametrize("order", (1, 2, 3))
def test_emulated_ranks_reproduce_the_single_domain(world, order):
    wl = W.CONFIGS["thermal_128"].scaled((16, 16, 32), shape_order=order, ppc=8, u_th=0.3)
    parts, fields = W.make_particles(wl), W.make_fields(wl)
    n_steps = 3
    ref = PP.gpu_for(wl, parts, fields)
    ref.step(n_steps)
    R = PP.gpu_particles_by_id(ref)
    Jr = ref.get_current().cpu().numpy().astype(np.float64)
    ref.destroy()

    dec = SL.SlabDecomposition(wl.grid, wl.cell, wl.supercell, world)
    make = lambda g: SL.PicStepper(g, wl.cell, wl.dt, wl.supercell, wl.shape_order)
    ranks = [SL.SlabRank(dec, r, make) for r in range(world)]
    gp = {k: getattr(parts, k).cuda() for k in ("x", "y", "z", "ux", "uy", "uz", "w", "species")}
    gp["gid"] = torch.arange(parts.n, dtype=torch.int64, device="cuda")
    f = fields.cuda()
    for r in ranks:
        r.take_owned(gp)
        r.set_global_fields(f)
    ex = SL.LoopbackExchange(dec)
    for _ in range(n_steps):
        SL.slab_step(ranks, ex)
    gids = torch.cat([r.parts["gid"] for r in ranks]).cpu().numpy()
    assert np.array_equal(np.sort(gids), np.arange(parts.n)), "particles lost or duplicated"
    for r in ranks:
        assert bool((dec.owner_of(r.parts["z"]) == r.rank).all())
        g = r.parts["gid"].cpu().numpy()
        for a, k in enumerate("xyz"):
            d = r.parts[k].cpu().numpy() - R[k][g]
            d -= wl.grid[a] * np.round(d / wl.grid[a])
            assert np.abs(d).max(initial=0.0) <= 1e-6, k       # same fp32 arithmetic on shifted coordinates
        for k in ("ux", "uy", "uz"):
            assert np.abs(r.parts[k].cpu().numpy() - R[k][g]).max(initial=0.0) <= 1e-6
        z0, z1 = dec.z_range(r.rank)
        assert np.abs(r.J.cpu().numpy() - Jr[:, z0:z1]).max() <= 2e-6 * np.abs(Jr).max()


@pytest.mark.parametrize("world", (2, 4))
def test_emulated_ranks_self_consistent_loop(world):
    """The same with the Yee update on every slab (pic_set_current with the exchanged J, pic_update_fields, E/B halo
    exchange) against the single-domain run with option field_update."""
    wl = W.CONFIGS["thermal_128"].scaled((16, 16, 32), shape_order=2, ppc=8, u_th=0.3)
    parts, fields = W.make_particles(wl), W.make_fields(wl)
    parts.w.mul_(0.01)
    n_steps = 3
    ref = PP.gpu_for(wl, parts, fields, field_update=1)
    ref.step(n_steps)
    R = PP.gpu_particles_by_id(ref)
    Jr = ref.get_current().cpu().numpy().astype(np.float64)
    Fr = ref.get_fields().cpu().numpy().astype(np.float64)
    ref.destroy()
    assert np.abs(Fr - fields.numpy()).max() > 0.02 * np.abs(Fr).max()

    dec = SL.SlabDecomposition(wl.grid, wl.cell, wl.supercell, world)
    make = lambda g: SL.PicStepper(g, wl.cell, wl.dt, wl.supercell, wl.shape_order)
    ranks = [SL.SlabRank(dec, r, make) for r in range(world)]
    gp = {k: getattr(parts, k).cuda() for k in ("x", "y", "z", "ux", "uy", "uz", "w", "species")}
    gp["gid"] = torch.arange(parts.n, dtype=torch.int64, device="cuda")
    f = fields.cuda()
    for r in ranks:
        r.take_owned(gp)
        r.set_global_fields(f)
    ex = SL.LoopbackExchange(dec)
    for _ in range(n_steps):
        SL.slab_step(ranks, ex, evolve_fields=True)
    gids = torch.cat([r.parts["gid"] for r in ranks]).cpu().numpy()
    assert np.array_equal(np.sort(gids), np.arange(parts.n))
    G = dec.guard
    for r in ranks:
        g = r.parts["gid"].cpu().numpy()
        for a, k in enumerate("xyz"):
            d = r.parts[k].cpu().numpy() - R[k][g]
            d -= wl.grid[a] * np.round(d / wl.grid[a])
            assert np.abs(d).max(initial=0.0) <= 2e-6, k
        for k in ("ux", "uy", "uz"):
            assert np.abs(r.parts[k].cpu().numpy() - R[k][g]).max(initial=0.0) <= 2e-6
        z0, z1 = dec.z_range(r.rank)
        assert np.abs(r.J.cpu().numpy() - Jr[:, z0:z1]).max() <= 5e-6 * np.abs(Jr).max()
        Fl = r.fields_local.cpu().numpy().astype(np.float64)
        assert np.abs(Fl[:, G:G + dec.owned_cells] - Fr[:, z0:z1]).max() <= 5e-6 * np.abs(Fr).max()
