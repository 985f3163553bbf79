"""Test-side helpers for the slab decomposition (tests only): a local stepper over the fp64 ORACLE with the five calls
slab.SlabRank expects, so that the exchange logic of paper_2110_08650_b200/slab.py can be held to the single-domain
oracle on CPU (gloo, world size 2) without a GPU."""
import numpy as np
import torch

import oracle


class OracleStepper:
    def __init__(self, grid, cell, dt, supercell, order):
        self.orc = oracle.Oracle(grid, cell, dt, supercell, order)
        self.n = 0

    def load(self, parts):
        self.n = int(parts["x"].numel())
        if self.n:
            self.orc.load_particles(*(parts[k].numpy() for k in ("x", "y", "z", "ux", "uy", "uz", "w")),
                                    species=parts["species"].numpy())

    def set_fields(self, fields):
        self.orc.set_fields(fields.numpy())

    def step(self):
        if self.n:
            assert self.orc.step(1) == 0

    def particles(self):
        P = self.orc.particles() if self.n else {k: np.zeros(0) for k in ("x", "y", "z", "ux", "uy", "uz", "w")}
        out = {k: torch.from_numpy(np.ascontiguousarray(P[k], dtype=np.float64)) for k in ("x", "y", "z")}
        for k in ("ux", "uy", "uz", "w"):
            out[k] = torch.from_numpy(np.ascontiguousarray(P[k], dtype=np.float64))      # kept in fp64: no rounding added
        out["species"] = torch.from_numpy(np.ascontiguousarray(self.orc.species if self.n else np.zeros(0, np.int32)))
        out["id"] = torch.arange(self.n, dtype=torch.int64)
        return out

    def current(self):
        return torch.from_numpy(np.stack(self.orc.J))

    def set_current(self, J):
        self.orc.J = tuple(np.ascontiguousarray(j, dtype=np.float64) for j in J.numpy())

    def update_fields(self):
        self.orc.update_fields()

    def fields(self):
        return torch.from_numpy(np.stack(self.orc.fields))


def global_particles(parts):
    """workloads.ParticleChunk -> dict with global ids."""
    d = {k: getattr(parts, k).clone() for k in ("x", "y", "z", "ux", "uy", "uz", "w", "species")}
    d["gid"] = torch.arange(parts.n, dtype=torch.int64)
    return d
