"""pic_deposit_current_noalloc (include/pic_b200.h): the entry point that allocates nothing — its scratch is a fixed
device array inside the library — against the EXISTING path (pic_create + workspace, pic_step, pic_get_current) on the
same particles: J within the J tolerance of the parity tests (1e-5 of max|J| after one step), on two calls in a row
with different inputs (the scratch array keeps the last call's sums: the second call must clear them itself).
Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest
import torch

import pic_parity as PP
from paper_2110_08650_b200 import binding
from paper_2110_08650_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _by_id(pic):
    P = pic.get_particles()
    order = torch.argsort(P["id"].to(torch.int64) & 0xFFFFFFFF)
    return {k: v[order].contiguous() for k, v in P.items()}


@pytest.mark.parametrize("order", (1, 2, 3))
def test_two_calls_in_a_row_match_the_existing_path(order):
    wl = W.CONFIGS["thermal_128"].scaled((32, 16, 16), shape_order=order, ppc=8, u_th=0.2)
    parts, fields = W.make_particles(wl), W.make_fields(wl)
    pic = PP.gpu_for(wl, parts, fields)
    states, currents = [_by_id(pic)], []
    for _ in range(2):
        pic.step(1)
        pic.sync()
        currents.append(pic.get_current().clone())
        states.append(_by_id(pic))
    assert pic.get_stats()["error"] == 0
    out = torch.full((3,) + tuple(wl.grid[::-1]), float("nan"), dtype=torch.float32, device="cuda")   # the CALLER's buffer
    for k in range(2):          # two calls in a row, different inputs, the same scratch array
        A, B = states[k], states[k + 1]
        qw = (-A["w"]).contiguous()              # default species: q = -1
        binding.deposit_current_noalloc(wl.grid, wl.cell, wl.dt, order, A["x"], A["y"], A["z"], B["x"], B["y"], B["z"],
                                        qw, out)
        torch.cuda.synchronize()
        ref = currents[k]
        scale = float(ref.abs().max())
        err = float((out - ref).abs().max())
        print(f"\n[no-alloc deposit, order {order}, call {k + 1}] err/max|J| = {err / scale:.3e}")
        assert scale > 0 and err <= PP.TOL_J1 * scale
    pic.destroy()


def test_limit_and_bad_moves_are_reported():
    dev = "cuda"
    z64 = torch.zeros(4, dtype=torch.float64, device=dev)
    qw = torch.ones(4, dtype=torch.float32, device=dev)
    big = (128, 64, 64)                                  # 524 288 cells > NOALLOC_MAX_CELLS
    assert big[0] * big[1] * big[2] > binding.NOALLOC_MAX_CELLS
    out = torch.empty((3, 64, 64, 128), dtype=torch.float32, device=dev)
    with pytest.raises(binding.PicError) as e:
        binding.deposit_current_noalloc(big, (1.0, 1.0, 1.0), 0.5, 2, z64, z64, z64, z64, z64, z64, qw, out)
    assert e.value.code == binding.PIC_EINVAL and "maximum" in str(e.value)
    # a move of a cell or more is not a step's move: left out, and flagged in the output
    out = torch.zeros((3, 8, 8, 8), dtype=torch.float32, device=dev)
    x0 = torch.tensor([1.25, 2.5, 3.0, 4.0], dtype=torch.float64, device=dev)
    x1 = x0.clone()
    x1[2] += 1.5
    binding.deposit_current_noalloc((8, 8, 8), (1.0, 1.0, 1.0), 0.5, 1, x0, x0, x0, x1, x0, x0, qw, out)
    torch.cuda.synchronize()
    assert bool(torch.isnan(out[:, 0, 0, 0]).all())
    # ... and the flag does not leak into the next call: particles at rest deposit exactly nothing
    binding.deposit_current_noalloc((8, 8, 8), (1.0, 1.0, 1.0), 0.5, 1, x0, x0, x0, x0, x0, x0, qw, out)
    torch.cuda.synchronize()
    assert float(out.abs().max()) == 0.0
