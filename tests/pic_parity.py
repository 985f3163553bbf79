"""Shared helpers of the CUDA-vs-oracle parity tests (tests only; imports both sides).

Tolerances are BASELINE.json:north_star's, read as SURVEY.md §8(c) S17, S18, S22:
  * positions: |dX| <= 2e-6 cells per step (min-image); momenta: |du| <= 2e-6 * max(|u|, u_scale) per step;
  * J: max|J_gpu - J_oracle| <= 1e-5 * max|J| after one step, 1e-4 after ten;
  * GPU continuity residual <= 1e-5 relative (rho from the GPU's own positions in fp64);
  * supercell counts / membership bit-exact, except particles whose oracle position lies within
    1e-6 cell (x number of free-running steps) of a supercell face, which are reported separately.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Dict, Optional

import numpy as np
import torch

import oracle
from paper_2110_08650_b200 import workloads as W

TOL_X = 2e-6
TOL_U = 2e-6
TOL_J1 = 1e-5
TOL_J10 = 1e-4
TOL_CONT = 1e-5
BAND = 1e-6


def oracle_for(wl: W.Workload, parts: W.ParticleChunk, fields: torch.Tensor) -> "oracle.Oracle":
    orc = oracle.Oracle(wl.grid, wl.cell, wl.dt, wl.supercell, wl.shape_order)
    orc.load_particles(*(getattr(parts, k).numpy() for k in ("x", "y", "z", "ux", "uy", "uz", "w")),
                       species=parts.species.numpy())
    orc.set_fields(fields.numpy())
    return orc


def gpu_for(wl: W.Workload, parts: W.ParticleChunk, fields: torch.Tensor, device="cuda:0", **options):
    from paper_2110_08650_b200.binding import Pic
    pic = Pic(wl.grid, wl.cell, wl.dt, wl.supercell, wl.shape_order, max_particles=parts.n, device=device)
    for k, v in options.items():
        pic.set_option(k, v)
    p = parts.to(device)
    pic.load_particles(p.x, p.y, p.z, p.ux, p.uy, p.uz, p.w, p.species)
    pic.set_fields(fields.to(device).contiguous())
    pic.sync()
    return pic


def gpu_particles_by_id(pic) -> Dict[str, np.ndarray]:
    P = pic.get_particles()
    ids = P["id"].to(torch.int64) & 0xFFFFFFFF
    order = torch.argsort(ids)
    out = {k: v[order].cpu().numpy() for k, v in P.items()}
    out["id"] = ids[order].cpu().numpy()
    return out


@dataclass
class ParityReport:
    n: int
    max_dx: float
    max_du_rel: float
    j_err_rel: float
    n_member_mismatch: int       # outside the band: must be 0
    n_near_face: int             # inside the band: reported separately (S18)
    n_near_face_mismatch: int
    counts_equal_outside_band: bool
    continuity: Optional[float] = None

    def __str__(self):
        return (f"n={self.n} max|dX|={self.max_dx:.3e} cells  max|du|/scale={self.max_du_rel:.3e}  "
                f"J err/max|J|={self.j_err_rel:.3e}  membership mismatches={self.n_member_mismatch} "
                f"(near-face particles {self.n_near_face}, of which differing {self.n_near_face_mismatch})"
                + (f"  continuity={self.continuity:.3e}" if self.continuity is not None else ""))


def compare(wl: W.Workload, orc: "oracle.Oracle", pic, n_steps: int, u_scale: float) -> ParityReport:
    """Element-by-element comparison after both sides advanced n_steps from the same state."""
    G = gpu_particles_by_id(pic)
    O = orc.particles()
    n = orc.n
    assert G["id"].size == n, f"particle count differs: gpu {G['id'].size} oracle {n}"
    assert np.array_equal(G["id"], np.arange(n)), "ids are not a permutation of the load order"
    assert np.array_equal(G["w"], O["w"].astype(np.float32)) and np.array_equal(G["species"], O["species"])
    max_dx = 0.0
    near = np.zeros(n, dtype=bool)
    for a, k in enumerate("xyz"):
        N = wl.grid[a]
        dX = (G[k] - O[k]) / wl.cell[a]
        dX -= N * np.round(dX / N)
        max_dx = max(max_dx, float(np.abs(dX).max()))
        Xo = O[k] / wl.cell[a]
        face = Xo / wl.supercell[a]
        dist = np.abs(face - np.round(face)) * wl.supercell[a]
        near |= dist <= BAND * n_steps
    du = np.sqrt(sum((G[k].astype(np.float64) - O[k]) ** 2 for k in ("ux", "uy", "uz")))
    un = np.sqrt(sum(O[k] ** 2 for k in ("ux", "uy", "uz")))
    max_du = float((du / np.maximum(un, u_scale)).max())
    mism = G["supercell"] != O["supercell"]
    Jg = pic.get_current().cpu().numpy().astype(np.float64)
    Jo = np.stack(orc.J)
    jmax = np.abs(Jo).max()
    j_err = float(np.abs(Jg - Jo).max() / jmax) if jmax > 0 else float(np.abs(Jg).max())
    # counts, with the near-face particles removed from both sides
    nsc = pic.n_supercells
    cg = np.bincount(G["supercell"][~near], minlength=nsc)
    co = np.bincount(O["supercell"][~near], minlength=nsc)
    counts_dev = pic.get_counts().cpu().numpy()
    assert np.array_equal(counts_dev, np.bincount(G["supercell"], minlength=nsc)), \
        "pic_get_counts disagrees with the membership pic_get_particles reports"
    return ParityReport(n, max_dx, max_du, j_err, int((mism & ~near).sum()), int(near.sum()),
                        int((mism & near).sum()), bool(np.array_equal(cg, co)))


def local_u_scale(wl: W.Workload, x, y, z, fields, n_steps: int, floor: float = 1e-3) -> np.ndarray:
    """S17 for the laser case, per particle: the momentum tolerance is relative to max(|u|, u_scale) with
    u_scale = |q/m| * F * dt/2, the momentum a particle at rest gains per step from the strongest field component F
    within reach (the 3^3 cells around its start, widened by one cell per further step) — a0*dt/2 = 0.5 at the
    centre of the pulse (reading D1), and the floor 1e-3 of S17 in the cold, field-free region."""
    F = torch.as_tensor(np.asarray(fields)).abs().amax(0)[None, None].to(torch.float32)      # [1,1,nz,ny,nx]
    r = n_steps
    Fp = torch.nn.functional.pad(F, (r, r, r, r, r, r), mode="circular")
    Fm = torch.nn.functional.max_pool3d(Fp, 2 * r + 1, stride=1)[0, 0].numpy()
    ci = [np.floor(np.asarray(c) / wl.cell[a]).astype(np.int64) % wl.grid[a] for a, c in enumerate((x, y, z))]
    return np.maximum(floor, 0.5 * wl.dt * Fm[ci[2], ci[1], ci[0]].astype(np.float64))


def gpu_membership_consistent(wl: W.Workload, pic) -> bool:
    """Membership reported by the library == floor(X) div SC recomputed from its own positions."""
    P = pic.get_particles()
    sc = wl.supercell
    nsx, nsy = wl.grid[0] // sc[0], wl.grid[1] // sc[1]
    c = [torch.floor(P[k] / wl.cell[a]).to(torch.int64) for a, k in enumerate("xyz")]
    for a in range(3):
        assert int(c[a].min()) >= 0 and int(c[a].max()) < wl.grid[a]
    exp = (c[0] // sc[0]) + nsx * ((c[1] // sc[1]) + nsy * (c[2] // sc[2]))
    return bool(torch.equal(exp.to(torch.int32), P["supercell"]))


def gpu_continuity(wl: W.Workload, pic, q_of_species) -> float:
    """S22: step the GPU once; rho^n, rho^{n+1} in fp64 (oracle.rho) from the GPU's own positions,
    div J from the GPU's J.  Returns max|drho/dt + div J| / max|drho/dt|."""
    prm = oracle.OracleParams.make(wl.grid, wl.cell, wl.dt, wl.supercell, wl.shape_order)
    A = gpu_particles_by_id(pic)
    pic.step(1)
    B = gpu_particles_by_id(pic)
    qw = np.asarray(q_of_species, dtype=np.float64)[A["species"]] * A["w"].astype(np.float64)
    cell = wl.cell
    rho0 = oracle.rho(prm, A["x"] / cell[0], A["y"] / cell[1], A["z"] / cell[2], qw)
    rho1 = oracle.rho(prm, B["x"] / cell[0], B["y"] / cell[1], B["z"] / cell[2], qw)
    Jx, Jy, Jz = pic.get_current().cpu().numpy().astype(np.float64)
    div = ((Jx - np.roll(Jx, 1, 2)) / cell[0] + (Jy - np.roll(Jy, 1, 1)) / cell[1]
           + (Jz - np.roll(Jz, 1, 0)) / cell[2])
    drho = (rho1 - rho0) / wl.dt
    return float(np.abs(drho + div).max() / np.abs(drho).max())


def energies(fields6, ux, uy, uz, w, cell, mass=1.0):
    """(electric, magnetic, kinetic) energy with c = eps0 = mu0 = 1: 1/2 sum F^2 dV and sum w m (gamma - 1).
    E, B at the integer time level, u at the half level before it (the state both sides hold)."""
    F = [np.asarray(f, dtype=np.float64) for f in fields6]
    V = cell[0] * cell[1] * cell[2]
    ef = 0.5 * V * sum(float((f * f).sum()) for f in F[:3])
    bf = 0.5 * V * sum(float((f * f).sum()) for f in F[3:6])
    u2 = np.asarray(ux, np.float64) ** 2 + np.asarray(uy, np.float64) ** 2 + np.asarray(uz, np.float64) ** 2
    ek = float((np.asarray(w, np.float64) * mass * (np.sqrt(1.0 + u2) - 1.0)).sum())
    return ef, bf, ek


def warm_dilute_plasma(order, grid=(16, 16, 16)):
    """Self-consistent test case: lambda_Debye = u_th/omega_p = 0.1/0.1 = one cell, field and kinetic energy of the
    same order, so the two reservoirs visibly exchange energy."""
    wl = W.CONFIGS["thermal_128"].scaled(grid, shape_order=order, ppc=8, u_th=0.1)
    parts, fields = W.make_particles(wl), W.make_fields(wl)
    parts.w.mul_(0.00125)
    return wl, parts, fields
