"""Slab decomposition: ownership, packing and the neighbour exchange of
paper_2110_08650_b200/slab.py, on CPU.  The local step is the fp64 oracle on the slab's local grid (guards included),
so the decomposed run must reproduce the single-domain oracle: every particle (by global id) to fp64 rounding of the
coordinate shift, J plane by plane, counts conserved.  World size 2 over gloo point-to-point calls, and the same
logic with the loop-back exchange for 1, 2 and 4 emulated ranks in one process."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

from paper_2110_08650_b200 import slab as SL                      # noqa: E402
from paper_2110_08650_b200 import workloads as W                  # noqa: E402


def _case(order=2, grid=(16, 16, 32), ppc=2, u_th=0.4):
    # fast particles: ~10 % cross a slab face in four steps, some across the periodic seam
    wl = W.CONFIGS["thermal_128"].scaled(grid, shape_order=order, ppc=ppc, u_th=u_th)
    return wl, W.make_particles(wl), W.make_fields(wl)


def _single_domain(wl, parts, fields, n_steps):
    import oracle
    orc = oracle.Oracle(wl.grid, wl.cell, wl.dt, wl.supercell, wl.shape_order)
    orc.load_particles(*(getattr(parts, k).numpy() for k in ("x", "y", "z", "ux", "uy", "uz", "w")),
                       species=parts.species.numpy())
    orc.set_fields(fields.numpy())
    assert orc.step(n_steps) == 0
    return orc.particles(), np.stack(orc.J)


def _check(wl, dec, ranks_state, ref_P, ref_J):
    """ranks_state: list of (rank, parts dict, J owned) gathered from all ranks."""
    n = ref_P["x"].size
    gids = np.concatenate([p["gid"].numpy() for _, p, _ in ranks_state])
    assert gids.size == n and np.array_equal(np.sort(gids), np.arange(n)), "particles lost or duplicated"
    for rank, p, J in ranks_state:
        assert bool((dec.owner_of(p["z"]) == rank).all()), "a rank holds a particle it does not own"
        g = p["gid"].numpy()
        for a, k in enumerate("xyz"):
            d = p[k].numpy() - ref_P[k][g]
            d -= wl.grid[a] * wl.cell[a] * np.round(d / (wl.grid[a] * wl.cell[a]))
            assert np.abs(d).max(initial=0.0) < 1e-11, k
        for k in ("ux", "uy", "uz"):
            assert np.abs(p[k].numpy().astype(np.float64) - ref_P[k][g]).max(initial=0.0) < 1e-12, k
        z0, z1 = dec.z_range(rank)
        assert np.abs(J.numpy() - ref_J[:, z0:z1]).max() <= 1e-12 * np.abs(ref_J).max()


@pytest.mark.parametrize("world", (1, 2, 4))
@pytest.mark.parametrize("order", (1, 2, 3))
def test_loopback_ranks_reproduce_the_single_domain(world, order):
    from slab_helpers import OracleStepper, global_particles
    wl, parts, fields = _case(order)
    n_steps = 4
    ref_P, ref_J = _single_domain(wl, parts, fields, n_steps)
    dec = SL.SlabDecomposition(wl.grid, wl.cell, wl.supercell, world)
    make = lambda g: OracleStepper(g, wl.cell, wl.dt, wl.supercell, wl.shape_order)
    ranks = [SL.SlabRank(dec, r, make, real=torch.float64) for r in range(world)]
    gp = global_particles(parts)
    for r in ranks:
        r.take_owned(gp)
        r.set_global_fields(fields.to(torch.float64))
    ex = SL.LoopbackExchange(dec)
    moved = 0
    for _ in range(n_steps):
        before = [set(r.parts["gid"].tolist()) for r in ranks]
        SL.slab_step(ranks, ex)
        moved += sum(len(set(r.parts["gid"].tolist()) - b) for r, b in zip(ranks, before))
    if world > 1:
        assert moved > 50, "the case must exercise the particle exchange"
    _check(wl, dec, [(r.rank, r.parts, r.J) for r in ranks], ref_P, ref_J)


def test_ownership_and_coordinates():
    dec = SL.SlabDecomposition((16, 16, 32), (1.0, 1.0, 0.5), (8, 8, 4), 4)
    assert dec.owned_cells == 8 and dec.local_grid == (16, 16, 16) and dec.z_range(3) == (24, 32)
    z = torch.tensor([0.0, 3.99, 4.0, 15.999, 16.0, -0.25, 16.25], dtype=torch.float64)     # cell size 0.5: domain [0,16)
    assert dec.owner_of(z).tolist() == [0, 0, 1, 3, 0, 3, 0]
    # rank 0: owned z in [0,4); a particle just below the seam sits in its low guard, one above its range in the high guard
    zl = dec.to_local_z(0, torch.tensor([15.75, 0.0, 3.5, 4.25], dtype=torch.float64))
    assert torch.allclose(zl, torch.tensor([1.75, 2.0, 5.5, 6.25], dtype=torch.float64))
    assert torch.allclose(dec.to_global_z(0, zl), torch.tensor([15.75, 0.0, 3.5, 4.25], dtype=torch.float64))
    f = torch.arange(32, dtype=torch.float64)[None, :, None, None].expand(6, 32, 2, 2)
    assert dec.local_fields(0, f)[0, :, 0, 0].tolist() == [28, 29, 30, 31] + list(range(0, 12))
    with pytest.raises(ValueError):
        SL.SlabDecomposition((16, 16, 32), (1, 1, 1), (8, 8, 4), 3)
    msg = SL.pack({k: torch.arange(5, dtype=torch.float64) for k in SL.KEYS}, torch.tensor([True, False, True, False, False]))
    assert msg.shape == (2, 9) and SL.unpack(msg)["gid"].tolist() == [0, 2]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from slab_helpers import OracleStepper, global_particles
    dist.init_process_group("gloo", rank=rank, world_size=world)
    wl, parts, fields = _case(2)
    dec = SL.SlabDecomposition(wl.grid, wl.cell, wl.supercell, world)
    me = SL.SlabRank(dec, rank, lambda g: OracleStepper(g, wl.cell, wl.dt, wl.supercell, wl.shape_order), real=torch.float64)
    me.take_owned(global_particles(parts))
    me.set_global_fields(fields.to(torch.float64))
    ex = SL.DistExchange(dec, rank)
    for _ in range(4):
        SL.slab_step([me], ex)
    dist.barrier()
    out[rank] = ({k: v.numpy() for k, v in me.parts.items()}, me.J.numpy())
    dist.destroy_process_group()


def test_two_processes_over_gloo():
    world = 2
    wl, parts, fields = _case(2)
    ref_P, ref_J = _single_domain(wl, parts, fields, 4)
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, 29547, out), nprocs=world, join=True)
        res = dict(out)
    dec = SL.SlabDecomposition(wl.grid, wl.cell, wl.supercell, world)
    state = [(r, {k: torch.from_numpy(v) for k, v in res[r][0].items()}, torch.from_numpy(res[r][1])) for r in range(world)]
    _check(wl, dec, state, ref_P, ref_J)


def _loop_case(order=2, grid=(16, 16, 32)):
    # a weakly coupled plasma (omega_p dt = 0.14) with fast particles: the fields visibly change and particles cross slabs
    wl = W.CONFIGS["thermal_128"].scaled(grid, shape_order=order, ppc=2, u_th=0.3)
    parts, fields = W.make_particles(wl), W.make_fields(wl)
    parts.w.mul_(0.04)
    return wl, parts, fields


def _single_domain_loop(wl, parts, fields, n_steps):
    import oracle
    orc = oracle.Oracle(wl.grid, wl.cell, wl.dt, wl.supercell, wl.shape_order)
    orc.load_particles(*(getattr(parts, k).numpy() for k in ("x", "y", "z", "ux", "uy", "uz", "w")),
                       species=parts.species.numpy())
    orc.set_fields(fields.numpy())
    assert orc.step(n_steps, update_fields=True) == 0
    return orc.particles(), np.stack(orc.J), np.stack(orc.fields)


def _check_fields(dec, ranks_fields, ref_F, ref_F0):
    scale = np.abs(ref_F).max()
    assert np.abs(ref_F - ref_F0).max() > 0.02 * scale, "the fields must have changed: this is not the static-field path"
    for rank, F in ranks_fields:
        z0, z1 = dec.z_range(rank)
        G = dec.guard
        assert np.abs(F[:, G:G + dec.owned_cells] - ref_F[:, z0:z1]).max() <= 1e-12 * scale
        # and the refreshed guards are the neighbours' planes
        idx = np.arange(z0 - G, z1 + G) % dec.grid[2]
        assert np.abs(F - ref_F[:, idx]).max() <= 1e-12 * scale


@pytest.mark.parametrize("world", (1, 2, 4))
def test_loopback_ranks_self_consistent_loop(world):
    """With the Yee update on every slab: J extended by the neighbours' edge planes, local update on slab + guards,
    E/B halo exchange.  Particles, J and fields against the single-domain self-consistent oracle."""
    from slab_helpers import OracleStepper, global_particles
    wl, parts, fields = _loop_case()
    n_steps = 4
    ref_P, ref_J, ref_F = _single_domain_loop(wl, parts, fields, n_steps)
    dec = SL.SlabDecomposition(wl.grid, wl.cell, wl.supercell, world)
    make = lambda g: OracleStepper(g, wl.cell, wl.dt, wl.supercell, wl.shape_order)
    ranks = [SL.SlabRank(dec, r, make, real=torch.float64) for r in range(world)]
    gp = global_particles(parts)
    for r in ranks:
        r.take_owned(gp)
        r.set_global_fields(fields.to(torch.float64))
    ex = SL.LoopbackExchange(dec)
    for _ in range(n_steps):
        SL.slab_step(ranks, ex, evolve_fields=True)
    _check(wl, dec, [(r.rank, r.parts, r.J) for r in ranks], ref_P, ref_J)
    _check_fields(dec, [(r.rank, r.fields_local.numpy()) for r in ranks], ref_F, fields.numpy().astype(np.float64))


def _worker_loop(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from slab_helpers import OracleStepper, global_particles
    dist.init_process_group("gloo", rank=rank, world_size=world)
    wl, parts, fields = _loop_case()
    dec = SL.SlabDecomposition(wl.grid, wl.cell, wl.supercell, world)
    me = SL.SlabRank(dec, rank, lambda g: OracleStepper(g, wl.cell, wl.dt, wl.supercell, wl.shape_order), real=torch.float64)
    me.take_owned(global_particles(parts))
    me.set_global_fields(fields.to(torch.float64))
    ex = SL.DistExchange(dec, rank)
    for _ in range(4):
        SL.slab_step([me], ex, evolve_fields=True)
    dist.barrier()
    out[rank] = ({k: v.numpy() for k, v in me.parts.items()}, me.J.numpy(), me.fields_local.numpy())
    dist.destroy_process_group()


def test_two_processes_over_gloo_self_consistent_loop():
    world = 2
    wl, parts, fields = _loop_case()
    ref_P, ref_J, ref_F = _single_domain_loop(wl, parts, fields, 4)
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker_loop, args=(world, 29549, out), nprocs=world, join=True)
        res = dict(out)
    dec = SL.SlabDecomposition(wl.grid, wl.cell, wl.supercell, world)
    state = [(r, {k: torch.from_numpy(v) for k, v in res[r][0].items()}, torch.from_numpy(res[r][1])) for r in range(world)]
    _check(wl, dec, state, ref_P, ref_J)
    _check_fields(dec, [(r, res[r][2]) for r in range(world)], ref_F, fields.numpy().astype(np.float64))
