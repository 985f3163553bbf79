"""Slab decomposition of the particle step over several GPUs.

The domain is cut along z into slabs of WHOLE supercell layers, one rank per slab.  A rank steps its slab on a local
grid that carries `guard` cells below and above the owned range (one supercell layer: the gather of a TSC/PQS
particle next to the slab face reads 2-3 cells beyond it, its Esirkepov current spills as far), then exchanges with
its two neighbours (periodic: rank 0 and rank W-1 are neighbours):

  1. particles whose new z left the owned range -> one packed message per neighbour (counts first, then payload);
  2. the current deposited into the guard planes -> added to the neighbour's outermost owned planes;
  3. (only when the fields evolve) the outermost owned E/B planes -> the neighbour's guard planes.

There is no all-reduce and nothing global: per step a rank sends ~1.5 % of its particles x 72 B and 2 x guard J planes.
NVSwitch makes every peer equidistant, so the slab order is arbitrary.

This module is the host logic: ownership, packing, the neighbour exchange over `torch.distributed` point-to-point
calls (NCCL on GPUs, gloo in the CPU tests) or, for several ranks emulated in ONE process, a loop-back exchange —
and `SlabRank`, which drives a local stepper (the CUDA library through `binding.Pic`, or any object with the same five
calls).  It holds none of the method's arithmetic.  State of the art here: correct by construction and tested at
world size 2 with gloo and, on one GPU, as emulated ranks against the single-domain run — static fields and the
self-consistent loop with the E/B halo exchange; no multi-GPU hardware was available to time it, and
`bench.py --gpus N` still runs replicas.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Callable, Dict, List, Optional, Sequence, Tuple

import torch

KEYS = ("x", "y", "z", "ux", "uy", "uz", "w", "species", "gid")


@dataclass(frozen=True)
class SlabDecomposition:
    grid: Tuple[int, int, int]          # global cells
    cell: Tuple[float, float, float]
    supercell: Tuple[int, int, int]
    world: int
    guard: int = 4                      # guard cells on either side (a whole supercell layer)

    def __post_init__(self):
        nz, scz = self.grid[2], self.supercell[2]
        if nz % scz or (nz // scz) % self.world:
            raise ValueError("the supercell layers along z must divide evenly among the ranks")
        if self.guard % scz or self.guard < scz:
            raise ValueError("guard must be a positive multiple of the supercell's z extent")
        if self.world > 1 and self.owned_cells < self.guard:
            raise ValueError("a slab must be at least as thick as the guard")

    @property
    def owned_cells(self) -> int:
        return self.grid[2] // self.world

    def z_range(self, rank: int) -> Tuple[int, int]:
        """Owned cells [z0, z1) of a rank."""
        return rank * self.owned_cells, (rank + 1) * self.owned_cells

    @property
    def local_grid(self) -> Tuple[int, int, int]:
        return (self.grid[0], self.grid[1], self.owned_cells + 2 * self.guard)

    def owner_of(self, z: torch.Tensor) -> torch.Tensor:
        """Rank that owns global position z (wrapped into the domain)."""
        L = self.grid[2] * self.cell[2]
        zc = torch.floor(torch.remainder(z, L) / self.cell[2]).to(torch.int64).clamp_(0, self.grid[2] - 1)
        return zc // self.owned_cells

    def to_local_z(self, rank: int, z: torch.Tensor) -> torch.Tensor:
        """Global z -> z on the rank's local grid (owned range starts at guard*cell); minimum image across the seam."""
        L = self.grid[2] * self.cell[2]
        z0 = self.z_range(rank)[0] * self.cell[2]
        rel = torch.remainder(z - z0, L)
        # owned range and the high guard stay as they are; what lies beyond them is below the slab (low guard)
        rel = torch.where(rel >= (self.owned_cells + self.guard) * self.cell[2], rel - L, rel)
        return rel + self.guard * self.cell[2]

    def to_global_z(self, rank: int, z_local: torch.Tensor) -> torch.Tensor:
        L = self.grid[2] * self.cell[2]
        z0 = self.z_range(rank)[0] * self.cell[2]
        return torch.remainder(z_local - self.guard * self.cell[2] + z0, L)

    def neighbours(self, rank: int) -> Tuple[int, int]:
        return (rank - 1) % self.world, (rank + 1) % self.world

    # ---------------------------------------------------------------- fields
    def local_fields(self, rank: int, fields: torch.Tensor) -> torch.Tensor:
        """[6 or 3, nz, ny, nx] global array -> the rank's local array with periodic guard planes."""
        z0, z1 = self.z_range(rank)
        idx = torch.arange(z0 - self.guard, z1 + self.guard, device=fields.device) % self.grid[2]
        return fields.index_select(1, idx).contiguous()


def pack(parts: Dict[str, torch.Tensor], sel: torch.Tensor) -> torch.Tensor:
    """Selected particles as one float64 [n, 9] message (positions are float64 at the boundary; ids < 2^53)."""
    return torch.stack([parts[k][sel].to(torch.float64) for k in KEYS], 1).contiguous()


def unpack(msg: torch.Tensor, real=torch.float32) -> Dict[str, torch.Tensor]:
    """The inverse of pack; `real` is the local stepper's type for momenta and weights (fp32 for the CUDA library)."""
    out = {}
    for i, k in enumerate(KEYS):
        col = msg[:, i]
        if k in ("x", "y", "z"):
            out[k] = col.clone()
        elif k == "species":
            out[k] = col.to(torch.int32)
        elif k == "gid":
            out[k] = col.to(torch.int64)
        else:
            out[k] = col.to(real)
    return out


def concat(a: Dict[str, torch.Tensor], b: Dict[str, torch.Tensor]) -> Dict[str, torch.Tensor]:
    return {k: torch.cat([a[k], b[k]]) for k in KEYS}


class DistExchange:
    """Neighbour exchange over torch.distributed point-to-point calls (one process per rank)."""

    def __init__(self, dec: SlabDecomposition, rank: int, group=None):
        import torch.distributed as dist
        self.dist, self.dec, self.rank, self.group = dist, dec, rank, group

    def _swap(self, to_lo: torch.Tensor, to_hi: torch.Tensor) -> Tuple[torch.Tensor, torch.Tensor]:
        """Send one tensor to each neighbour, receive one from each: sizes first, then payloads.  Returns
        (from_lo, from_hi).  With world size 2 both neighbours are the same rank: the two directions are kept apart
        by their order (up-going first)."""
        dist, (lo, hi) = self.dist, self.dec.neighbours(self.rank)
        dev = to_lo.device
        cols = to_lo.shape[1:]
        n_out = torch.tensor([to_hi.shape[0], to_lo.shape[0]], dtype=torch.int64, device=dev)
        n_in = torch.zeros(2, dtype=torch.int64, device=dev)
        # up-going: send to hi, receive from lo; then down-going: send to lo, receive from hi
        ops = [dist.P2POp(dist.isend, n_out[0:1], hi, self.group), dist.P2POp(dist.irecv, n_in[0:1], lo, self.group)]
        for r in dist.batch_isend_irecv(ops):
            r.wait()
        ops = [dist.P2POp(dist.isend, n_out[1:2], lo, self.group), dist.P2POp(dist.irecv, n_in[1:2], hi, self.group)]
        for r in dist.batch_isend_irecv(ops):
            r.wait()
        from_lo = torch.empty((int(n_in[0]),) + tuple(cols), dtype=to_lo.dtype, device=dev)
        from_hi = torch.empty((int(n_in[1]),) + tuple(cols), dtype=to_lo.dtype, device=dev)
        ops = []
        if to_hi.shape[0]:
            ops.append(dist.P2POp(dist.isend, to_hi.contiguous(), hi, self.group))
        if from_lo.shape[0]:
            ops.append(dist.P2POp(dist.irecv, from_lo, lo, self.group))
        if ops:
            for r in dist.batch_isend_irecv(ops):
                r.wait()
        ops = []
        if to_lo.shape[0]:
            ops.append(dist.P2POp(dist.isend, to_lo.contiguous(), lo, self.group))
        if from_hi.shape[0]:
            ops.append(dist.P2POp(dist.irecv, from_hi, hi, self.group))
        if ops:
            for r in dist.batch_isend_irecv(ops):
                r.wait()
        return from_lo, from_hi

    def swap_all(self, outgoing: Sequence[Tuple[torch.Tensor, torch.Tensor]]):
        return [self._swap(*outgoing[0])]


class LoopbackExchange:
    """All ranks in one process (tests on a single GPU): swap_all takes every rank's (to_lo, to_hi) at once."""

    def __init__(self, dec: SlabDecomposition):
        self.dec = dec

    def swap_all(self, outgoing: Sequence[Tuple[torch.Tensor, torch.Tensor]]):
        W = self.dec.world
        return [(outgoing[(r - 1) % W][1], outgoing[(r + 1) % W][0]) for r in range(W)]


class PicStepper:
    """Local stepper over the CUDA library: one fresh context per step (the C ABI has no call that removes particles;
    a production path would hand the library's exchange buffer to the neighbour instead of reading everything back)."""

    def __init__(self, grid, cell, dt, supercell, shape_order, device="cuda:0", **options):
        self.args, self.device, self.options = (grid, cell, dt, supercell, shape_order), device, options
        self.pic = None

    def load(self, parts: Dict[str, torch.Tensor]):
        from .binding import Pic
        if self.pic is not None:
            self.pic.destroy()
        n = int(parts["x"].numel())
        self.pic = Pic(*self.args, max_particles=max(n, 1), device=self.device)
        for k, v in self.options.items():
            self.pic.set_option(k, v)
        d = self.device
        if n:
            self.pic.load_particles(*(parts[k].to(d) for k in ("x", "y", "z", "ux", "uy", "uz", "w", "species")))
        self.n = n

    def set_fields(self, fields: torch.Tensor):
        self.pic.set_fields(fields.to(self.device).contiguous())

    def step(self):
        if self.n:
            self.pic.step(1)

    def particles(self) -> Dict[str, torch.Tensor]:
        if not self.n:
            z = torch.zeros(0, dtype=torch.float64, device=self.device)
            return {**{k: z for k in "xyz"}, **{k: z.to(torch.float32) for k in ("ux", "uy", "uz", "w")},
                    "species": z.to(torch.int32), "id": z.to(torch.int64)}
        P = self.pic.get_particles()
        P["id"] = P["id"].to(torch.int64) & 0xFFFFFFFF
        return P

    def current(self) -> torch.Tensor:
        if not self.n:
            g = self.args[0]
            return torch.zeros((3, g[2], g[1], g[0]), dtype=torch.float32, device=self.device)
        return self.pic.get_current()

    # ---- evolving fields: the completed J goes back in before the Yee update (pic_set_current)
    def set_current(self, J: torch.Tensor):
        self.pic.set_current(J.to(self.device, torch.float32).contiguous())

    def update_fields(self):
        self.pic.update_fields()

    def fields(self) -> torch.Tensor:
        return self.pic.get_fields()


class SlabRank:
    """One rank's share of the domain: its particles (global coordinates, global ids) and its owned planes of J."""

    def __init__(self, dec: SlabDecomposition, rank: int, make_stepper: Callable[[Tuple[int, int, int]], object],
                 real=torch.float32):
        self.dec, self.rank, self.make_stepper, self.real = dec, rank, make_stepper, real
        self.parts: Optional[Dict[str, torch.Tensor]] = None
        self.J: Optional[torch.Tensor] = None          # [3, owned, ny, nx]
        self.fields_local: Optional[torch.Tensor] = None
        self._J_local = None

    def take_owned(self, parts: Dict[str, torch.Tensor]):
        """Keep the particles of a global set that this rank owns (parts has a 'gid' entry)."""
        own = self.dec.owner_of(parts["z"]) == self.rank
        self.parts = {k: parts[k][own] for k in KEYS}

    def set_global_fields(self, fields: torch.Tensor):
        self.fields_local = self.dec.local_fields(self.rank, fields)

    # ---- the three phases of a step
    def local_step(self):
        dec, p = self.dec, self.parts
        local = dict(p)
        local["z"] = dec.to_local_z(self.rank, p["z"])
        st = self.make_stepper(dec.local_grid)
        st.load(local)
        st.set_fields(self.fields_local)
        st.step()
        P = st.particles()
        order = P["id"].to(torch.int64)
        gid = p["gid"].to(order.device)[order]
        self.parts = {k: P[k] for k in ("x", "y", "ux", "uy", "uz", "w", "species")}
        self.parts["z"] = dec.to_global_z(self.rank, P["z"])
        self.parts["gid"] = gid
        self._J_local = st.current()
        self._st = st

    def outgoing_particles(self) -> Tuple[torch.Tensor, torch.Tensor]:
        dec = self.dec
        owner = dec.owner_of(self.parts["z"])
        lo, hi = dec.neighbours(self.rank)
        stay = owner == self.rank
        # with two ranks both neighbours are the same rank: direction decides (a leaver crossed the nearer face)
        zl = dec.to_local_z(self.rank, self.parts["z"])
        below = (~stay) & (zl < dec.guard * dec.cell[2])
        above = (~stay) & ~below
        msgs = pack(self.parts, below), pack(self.parts, above)
        self.parts = {k: self.parts[k][stay] for k in KEYS}
        return msgs

    def incoming_particles(self, from_lo: torch.Tensor, from_hi: torch.Tensor):
        inc = unpack(torch.cat([from_lo, from_hi]), self.real)
        self.parts = concat(self.parts, {k: inc[k].to(self.parts[k].device) for k in KEYS})

    def outgoing_current(self) -> Tuple[torch.Tensor, torch.Tensor]:
        G, own = self.dec.guard, self.dec.owned_cells
        J = self._J_local
        self.J = J[:, G:G + own].clone()
        return (J[:, :G].permute(1, 0, 2, 3).contiguous(), J[:, G + own:].permute(1, 0, 2, 3).contiguous())

    def incoming_current(self, from_lo: torch.Tensor, from_hi: torch.Tensor):
        G, own = self.dec.guard, self.dec.owned_cells
        self.J[:, :G] += from_lo.permute(1, 0, 2, 3).to(self.J.device)
        self.J[:, own - G:] += from_hi.permute(1, 0, 2, 3).to(self.J.device)


def _owned_edge_planes(A: torch.Tensor, dec: SlabDecomposition) -> Tuple[torch.Tensor, torch.Tensor]:
    """A: [C, owned, ny, nx] -> (bottom G planes for the lower neighbour, top G planes for the upper one), planes first."""
    G = dec.guard
    return A[:, :G].permute(1, 0, 2, 3).contiguous(), A[:, -G:].permute(1, 0, 2, 3).contiguous()


def _with_guards(A: torch.Tensor, from_lo: torch.Tensor, from_hi: torch.Tensor) -> torch.Tensor:
    """Owned planes + the neighbours' edge planes as guards: [C, G + owned + G, ny, nx]."""
    return torch.cat([from_lo.permute(1, 0, 2, 3).to(A.device, A.dtype), A, from_hi.permute(1, 0, 2, 3).to(A.device, A.dtype)], 1).contiguous()


def slab_step(ranks: List[SlabRank], exchange, evolve_fields: bool = False) -> None:
    """One step of every rank in `ranks` (one entry with DistExchange, all ranks with LoopbackExchange).
    evolve_fields: the step ends with the Yee update of E, B on every slab: the completed J is
    extended by the neighbours' edge planes (the update of an owned cell reads J, E, B up to two cells away: less than
    the guard), the local update runs on slab + guards, and the guards of the new E, B are refreshed from the
    neighbours' owned planes — the E/B halo exchange."""
    for r in ranks:
        r.local_step()
    inc = exchange.swap_all([r.outgoing_particles() for r in ranks])
    for r, (flo, fhi) in zip(ranks, inc):
        r.incoming_particles(flo, fhi)
    inc = exchange.swap_all([r.outgoing_current() for r in ranks])
    for r, (flo, fhi) in zip(ranks, inc):
        r.incoming_current(flo, fhi)
    if not evolve_fields:
        return
    dec = ranks[0].dec
    G, own = dec.guard, dec.owned_cells
    inc = exchange.swap_all([_owned_edge_planes(r.J, dec) for r in ranks])
    for r, (flo, fhi) in zip(ranks, inc):
        r._st.set_current(_with_guards(r.J, flo, fhi))
        r._st.update_fields()
        r._F_owned = r._st.fields()[:, G:G + own].clone()
    inc = exchange.swap_all([_owned_edge_planes(r._F_owned, dec) for r in ranks])
    for r, (flo, fhi) in zip(ranks, inc):
        r.fields_local = _with_guards(r._F_owned, flo, fhi)
