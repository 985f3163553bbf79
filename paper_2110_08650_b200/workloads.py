"""Seeded synthetic inputs for the PIC particle step (BASELINE.json:configs).

This module is the ONLY thing shared between the CUDA path and the CPU oracle: it
holds no arithmetic of the method (no shape functions, no push, no deposit) — only
the recipes that draw positions, momenta, weights and the external E/B fields.  The
same arrays it returns are handed to both sides, so RNG reproducibility across
implementations is never needed.

Exchange format: positions are float64 in cell units times the
cell size, built as ``integer cell + float32 in-cell fraction`` so that they are
exactly representable both as float64 and as (cell, fp32 fraction); momenta
``u = gamma*beta`` and weights are float32; species is int32.

Field arrays are float32 ``[nz, ny, nx]`` (C order == index ``i + nx*(j + ny*k)``)
sampled at the Yee location of each component.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import Dict, Iterator, Optional, Tuple

import torch

# Yee stagger (in cells) of Ex,Ey,Ez,Bx,By,Bz along (x,y,z): SURVEY.md §8(c) step 2.
YEE_STAGGER = (
    (0.5, 0.0, 0.0),
    (0.0, 0.5, 0.0),
    (0.0, 0.0, 0.5),
    (0.0, 0.5, 0.5),
    (0.5, 0.0, 0.5),
    (0.5, 0.5, 0.0),
)


@dataclass(frozen=True)
class Workload:
    """One entry of BASELINE.json:configs (readings S5-S13 of SURVEY.md §8(c))."""

    name: str
    grid: Tuple[int, int, int]
    shape_order: int                      # 1 CIC, 2 TSC, 3 PQS
    ppc: int
    seed: int
    steps: int
    u_th: float = 0.0
    dt: float = 0.5                       # S5
    cell: Tuple[float, float, float] = (1.0, 1.0, 1.0)
    supercell: Tuple[int, int, int] = (8, 8, 4)
    fields: str = "uniform"               # uniform | modes | laser
    n_modes: int = 8
    amplitude: float = 0.01
    uniform_E: Tuple[float, float, float] = (0.01, 0.0, 0.0)
    uniform_B: Tuple[float, float, float] = (0.0, 0.0, 0.1)
    layout: str = "uniform"               # uniform | slab_ramp | two_stream | hotspot
    drift_beta: float = 0.0               # two_stream: +-beta_y (S8)
    slab_y0_frac: float = 0.25            # slab_ramp: plasma in y >= y0 (S13: 256/1024)
    ramp_cells: int = 64
    hot_fraction: float = 0.5             # hotspot (S11)
    hot_supercell_fraction: float = 0.01
    laser: Dict[str, float] = field(default_factory=dict)

    @property
    def n_cells(self) -> int:
        return self.grid[0] * self.grid[1] * self.grid[2]

    def scaled(self, grid: Tuple[int, int, int], name: Optional[str] = None, **kw) -> "Workload":
        """Same recipe on a smaller grid (reduced-size parity tier T2 of SURVEY.md §8(d))."""
        return replace(self, grid=tuple(grid), name=name or f"{self.name}@{grid[0]}x{grid[1]}x{grid[2]}", **kw)


CONFIGS: Dict[str, Workload] = {
    # configs[0]
    "tiny_thermal": Workload("tiny_thermal", (16, 16, 16), 1, 8, 0, 10, u_th=0.01, fields="uniform"),
    # configs[1] — the config the metric is quoted on
    "thermal_128": Workload("thermal_128", (128, 128, 128), 2, 16, 1, 100, u_th=0.05,
                            fields="modes", n_modes=8, amplitude=0.01),
    # configs[2]
    "lwfa": Workload("lwfa", (256, 1024, 256), 2, 2, 2, 50, u_th=0.0, fields="laser",
                     layout="slab_ramp",
                     laser=dict(a0=2.0, w0=32.0, w_y=16.0, wavelength=16.0, y0_frac=0.375)),
    # configs[3] (+ hot-spot variant)
    "khi": Workload("khi", (192, 192, 192), 2, 9, 3, 100, u_th=0.01, fields="modes",
                    n_modes=8, amplitude=0.01, layout="two_stream", drift_beta=0.2),
    "khi_hotspot": Workload("khi_hotspot", (192, 192, 192), 2, 9, 3, 100, u_th=0.01,
                            fields="modes", n_modes=8, amplitude=0.01, layout="hotspot",
                            drift_beta=0.2),
    # configs[4]
    "pqs_large": Workload("pqs_large", (512, 512, 256), 3, 8, 4, 20, u_th=0.1,
                          fields="modes", n_modes=16, amplitude=0.05),
}


def _gen(seed: int, stream: int, device) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed((int(seed) * 1_000_003 + int(stream) * 7919 + 12345) & 0x7FFFFFFFFFFF)
    return g


# --------------------------------------------------------------------------- fields
def make_fields(wl: Workload, device="cpu") -> torch.Tensor:
    """float32 tensor [6, nz, ny, nx]: Ex,Ey,Ez,Bx,By,Bz at their Yee locations."""
    nx, ny, nz = wl.grid
    out = torch.zeros((6, nz, ny, nx), dtype=torch.float32, device=device)
    if wl.fields == "uniform":
        for c in range(3):
            out[c].fill_(wl.uniform_E[c])
            out[3 + c].fill_(wl.uniform_B[c])
        return out
    # node coordinates in cells (float64 for the phase, result rounded to fp32)
    ax = [torch.arange(n, dtype=torch.float64, device=device) for n in (nx, ny, nz)]
    if wl.fields == "modes":
        # S12: F_c(r) = sum_m (A/M) cos(2 pi k_m.r/N + phi_{m,c}), k_m in {-4..4}^3 \ {0}
        gk = _gen(wl.seed, 101, "cpu")
        M = wl.n_modes
        ks = []
        while len(ks) < M:
            k = torch.randint(-4, 5, (3,), generator=gk)
            if int(k.abs().sum()) != 0:
                ks.append(k)
        phis = torch.rand((M, 6), generator=gk, dtype=torch.float64) * (2.0 * math.pi)
        for c in range(6):
            sx, sy, sz = YEE_STAGGER[c]
            acc = torch.zeros((nz, ny, nx), dtype=torch.float64, device=device)
            for m in range(M):
                kx, ky, kz = (int(v) for v in ks[m])
                px = 2.0 * math.pi * kx * (ax[0] + sx) / nx
                py = 2.0 * math.pi * ky * (ax[1] + sy) / ny
                pz = 2.0 * math.pi * kz * (ax[2] + sz) / nz
                acc += torch.cos(pz[:, None, None] + py[None, :, None] + px[None, None, :] + float(phis[m, c]))
            out[c] = (acc * (wl.amplitude / M)).to(torch.float32)
        return out
    if wl.fields == "laser":
        # S13 (y0: DESIGN.md reading D6 — inside the plasma, the static pulse would otherwise touch no particle):
        # E_x = a0 exp(-((y-y0)/w_y)^2 - ((x-xc)^2+(z-zc)^2)/w0^2) cos(k (y-y0)), B_z = E_x,
        # each evaluated at its own Yee location; all other components 0.
        L = wl.laser
        xc, zc = nx / 2.0, nz / 2.0
        y0 = L["y0_frac"] * ny
        k = 2.0 * math.pi / L["wavelength"]
        for c in (0, 5):
            sx, sy, sz = YEE_STAGGER[c]
            X = ax[0] + sx - xc
            Y = ax[1] + sy - y0
            Z = ax[2] + sz - zc
            env_y = torch.exp(-(Y / L["w_y"]) ** 2) * torch.cos(k * Y)
            env_x = torch.exp(-(X / L["w0"]) ** 2)
            env_z = torch.exp(-(Z / L["w0"]) ** 2)
            out[c] = (L["a0"] * env_z[:, None, None] * env_y[None, :, None] * env_x[None, None, :]).to(torch.float32)
        return out
    raise ValueError(f"unknown field recipe {wl.fields!r}")


# ------------------------------------------------------------------------ particles
@dataclass
class ParticleChunk:
    x: torch.Tensor        # float64 [n] global position (cell + fp32 fraction) * cell size
    y: torch.Tensor
    z: torch.Tensor
    ux: torch.Tensor       # float32 [n] gamma*beta
    uy: torch.Tensor
    uz: torch.Tensor
    w: torch.Tensor        # float32 [n]
    species: torch.Tensor  # int32 [n]

    @property
    def n(self) -> int:
        return int(self.x.numel())

    def to(self, device) -> "ParticleChunk":
        return ParticleChunk(*(getattr(self, k).to(device) for k in
                               ("x", "y", "z", "ux", "uy", "uz", "w", "species")))

    @staticmethod
    def cat(chunks) -> "ParticleChunk":
        chunks = list(chunks)
        return ParticleChunk(*(torch.cat([getattr(c, k) for c in chunks]) for k in
                               ("x", "y", "z", "ux", "uy", "uz", "w", "species")))


def n_particles(wl: Workload) -> int:
    nx, ny, nz = wl.grid
    if wl.layout == "slab_ramp":
        y0 = int(round(wl.slab_y0_frac * ny))
        return nx * (ny - y0) * nz * wl.ppc
    return wl.n_cells * wl.ppc


def _hot_supercells(wl: Workload) -> torch.Tensor:
    nsx, nsy, nsz = (wl.grid[a] // wl.supercell[a] for a in range(3))
    nsc = nsx * nsy * nsz
    n_hot = max(1, int(math.floor(wl.hot_supercell_fraction * nsc)))
    g = _gen(wl.seed, 202, "cpu")
    return torch.randperm(nsc, generator=g)[:n_hot].sort().values


def _cells_to_particles(wl: Workload, ci, cj, ck, chunk_id: int, device) -> ParticleChunk:
    """ci,cj,ck: int64 cell indices, one entry per particle."""
    n = ci.numel()
    g = _gen(wl.seed, 1000 + chunk_id, device)
    frac = torch.rand((3, n), generator=g, dtype=torch.float32, device=device)   # [0,1) fp32
    X = [(c.to(torch.float64) + frac[a].to(torch.float64)) * wl.cell[a] for a, c in enumerate((ci, cj, ck))]
    if wl.u_th > 0.0:
        u = torch.randn((3, n), generator=g, dtype=torch.float32, device=device) * wl.u_th   # S7
    else:
        u = torch.zeros((3, n), dtype=torch.float32, device=device)
    w = torch.ones(n, dtype=torch.float32, device=device)
    species = torch.zeros(n, dtype=torch.int32, device=device)
    nx, ny, nz = wl.grid
    if wl.layout in ("two_stream", "hotspot"):
        # S8/S9: species 0 (+drift) fills x in [nx/4, 3nx/4), species 1 (-drift) the outer quarters
        inner = (ci >= nx // 4) & (ci < (3 * nx) // 4)
        species = torch.where(inner, 0, 1).to(torch.int32)
        u_d = wl.drift_beta / math.sqrt(1.0 - wl.drift_beta ** 2)
        u[1] += torch.where(inner, u_d, -u_d).to(torch.float32)
    if wl.layout == "slab_ramp":
        y0 = int(round(wl.slab_y0_frac * ny))
        yy = cj.to(torch.float64) + frac[1].to(torch.float64)
        w = torch.clamp((yy - y0) / wl.ramp_cells, max=1.0).to(torch.float32)   # S13
    return ParticleChunk(X[0], X[1], X[2], u[0].contiguous(), u[1].contiguous(), u[2].contiguous(), w, species)


def particle_chunks(wl: Workload, device="cpu", max_chunk: int = 1 << 24) -> Iterator[ParticleChunk]:
    """Yield the workload's particles in chunks of whole z-slabs (<= ~max_chunk particles)."""
    nx, ny, nz = wl.grid
    if wl.layout == "hotspot":
        yield from _hotspot_chunks(wl, device, max_chunk)
        return
    y_lo = int(round(wl.slab_y0_frac * ny)) if wl.layout == "slab_ramp" else 0
    per_slab = nx * (ny - y_lo) * wl.ppc
    slabs = max(1, min(nz, max_chunk // max(per_slab, 1)))
    ii = torch.arange(nx, device=device)
    jj = torch.arange(y_lo, ny, device=device)
    for cid, z0 in enumerate(range(0, nz, slabs)):
        kk = torch.arange(z0, min(nz, z0 + slabs), device=device)
        K, J, I = torch.meshgrid(kk, jj, ii, indexing="ij")
        ci = I.reshape(-1).repeat_interleave(wl.ppc)
        cj = J.reshape(-1).repeat_interleave(wl.ppc)
        ck = K.reshape(-1).repeat_interleave(wl.ppc)
        yield _cells_to_particles(wl, ci, cj, ck, cid, device)


def _hotspot_chunks(wl: Workload, device, max_chunk: int) -> Iterator[ParticleChunk]:
    """S11: hot_fraction of all particles uniformly inside 1% of the supercells, the rest
    uniformly over the other supercells."""
    nx, ny, nz = wl.grid
    scx, scy, scz = wl.supercell
    nsx, nsy, nsz = nx // scx, ny // scy, nz // scz
    nsc = nsx * nsy * nsz
    hot = _hot_supercells(wl).to(device)
    is_hot = torch.zeros(nsc, dtype=torch.bool, device=device)
    is_hot[hot] = True
    cold = torch.nonzero(~is_hot).reshape(-1)
    n_total = n_particles(wl)
    n_hot_p = int(wl.hot_fraction * n_total)
    parts = [(hot, n_hot_p), (cold, n_total - n_hot_p)]
    cid = 0
    for scs, n_p in parts:
        done = 0
        while done < n_p:
            n = min(max_chunk, n_p - done)
            g = _gen(wl.seed, 5000 + cid, device)
            pick = scs[torch.randint(0, scs.numel(), (n,), generator=g, device=device)]
            sx = pick % nsx
            sy = (pick // nsx) % nsy
            sz = pick // (nsx * nsy)
            loc = torch.randint(0, scx * scy * scz, (n,), generator=g, device=device)
            ci = sx * scx + loc % scx
            cj = sy * scy + (loc // scx) % scy
            ck = sz * scz + loc // (scx * scy)
            yield _cells_to_particles(wl, ci, cj, ck, 100 + cid, device)
            done += n
            cid += 1


def make_particles(wl: Workload, device="cpu") -> ParticleChunk:
    """All particles at once (small / reduced-size workloads)."""
    return ParticleChunk.cat(particle_chunks(wl, device))
