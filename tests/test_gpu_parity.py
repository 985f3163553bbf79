"""CUDA-vs-oracle parity of the PIC particle step, through the C ABI (binding.Pic).

Cases: configs[0] at full size (1 and 10 steps) and reduced-grid copies of configs[1..4]
(same ppc, shape order, field recipe; SURVEY.md §8(d) tier T2), each spanning several
supercells, several frames per supercell and a ragged last frame.  Tolerances: tests/pic_parity.py.
"""
import numpy as np
import pytest
import torch

import pic_parity as PP
from paper_2110_08650_b200 import workloads as W

pytestmark = pytest.mark.gpu

CASES = {
    # name: (workload, u_scale for the momentum tolerance (S17))
    "cfg1_tiny_cic": (W.CONFIGS["tiny_thermal"], 0.01),
    "cfg2_thermal_tsc_32": (W.CONFIGS["thermal_128"].scaled((32, 32, 32)), 0.05),
    # S17: momentum scale of the laser case, per particle from the field within its reach: a0 * |q/m| * dt/2 = 0.5 at
    # the pulse centre, 1e-3 in the cold region (pic_parity.local_u_scale)
    "cfg3_lwfa_tsc_32x128x32": (W.CONFIGS["lwfa"].scaled((32, 128, 32)), "local"),
    "cfg4_khi_tsc_24": (W.CONFIGS["khi"].scaled((24, 24, 24)), 0.01),
    "cfg4_khi_hotspot_tsc_24": (W.CONFIGS["khi_hotspot"].scaled((24, 24, 24)), 0.01),
    "cfg5_pqs_32x32x16": (W.CONFIGS["pqs_large"].scaled((32, 32, 16)), 0.1),
}


def _run(name, n_steps, **options):
    wl, u_scale = CASES[name]
    parts, fields = W.make_particles(wl), W.make_fields(wl)
    orc = PP.oracle_for(wl, parts, fields)
    pic = PP.gpu_for(wl, parts, fields, **options)
    if u_scale == "local":
        u_scale = PP.local_u_scale(wl, parts.x.numpy(), parts.y.numpy(), parts.z.numpy(), fields.numpy(), n_steps)
    assert orc.step(n_steps) == 0
    pic.step(n_steps)
    pic.sync()
    rep = PP.compare(wl, orc, pic, n_steps, u_scale)
    print(f"\n[{name} steps={n_steps} {options}] {rep}")
    st = pic.get_stats()
    assert st["error"] == 0 and st["particles"] == parts.n and st["steps"] == n_steps
    assert PP.gpu_membership_consistent(wl, pic)
    return rep, pic, wl


@pytest.mark.parametrize("name", list(CASES))
@pytest.mark.parametrize("tma", (0, 1))
def test_one_step(name, tma):
    rep, pic, wl = _run(name, 1, tma=tma)
    assert rep.max_dx <= PP.TOL_X
    assert rep.max_du_rel <= PP.TOL_U
    assert rep.j_err_rel <= PP.TOL_J1
    assert rep.n_member_mismatch == 0 and rep.counts_equal_outside_band
    pic.destroy()


@pytest.mark.parametrize("name", list(CASES))
@pytest.mark.parametrize("kernel", (0, 1, 2))
def test_dense_kernel_generations(name, kernel):
    """Option cell_kernel: 0 the round-1 dense kernels (work items of <= LMAX particles), 1 pic_cell_kernel (one CTA
    per supercell, one thread per cell), 2 pic_pcell_kernel (persistent CTAs, producer warps sort and stage the
    next supercell beside the consumer warps).  Each is held to the oracle for three free-running steps (the second
    and third start from a fused sort of the stepped state)."""
    rep, pic, wl = _run(name, 3, cell_kernel=kernel)
    assert rep.max_dx <= 3 * PP.TOL_X and rep.max_du_rel <= 3 * PP.TOL_U and rep.j_err_rel <= PP.TOL_J10
    assert rep.n_member_mismatch == 0 and rep.counts_equal_outside_band
    pic.destroy()


def test_particles_at_rest_in_field_free_supercells_are_skipped_exactly():
    """configs[2] shape: cold plasma (u = 0 exactly) and a laser pulse that underflows to exact zeros away from its
    centre.  The one-thread-per-particle variant skips warps of particles at rest in supercells whose E/B tile is all
    zero (option rest_skip, default on); with the option off every particle is stepped.  Positions, momenta and J after 6
    steps must agree bit for bit (J in fixed point, sparse_float = 0: the float accumulation of all-sparse steps depends
    on the order of its atomics), and the case must contain both kinds of particle."""
    wl = W.CONFIGS["lwfa"].scaled((16, 512, 8))      # long enough along y for the pulse (w_y = 16 cells) to die out
    parts, fields = W.make_particles(wl), W.make_fields(wl)
    assert float(parts.ux.abs().max()) == 0.0 and float(parts.uy.abs().max()) == 0.0     # cold start
    nz_planes = (fields.abs().amax(dim=(0, 1, 3)) > 0).sum().item()
    assert 0 < nz_planes < wl.grid[1] - 16          # the pulse covers part of y only: field-free supercells exist
    out = []
    for skip in (1, 0):
        pic = PP.gpu_for(wl, parts, fields, rest_skip=skip, sparse_float=0)
        pic.step(6)
        pic.sync()
        assert pic.get_stats()["error"] == 0
        out.append((PP.gpu_particles_by_id(pic), pic.get_current().cpu()))
        pic.destroy()
    (A, JA), (B, JB) = out
    for k in ("x", "y", "z", "ux", "uy", "uz"):
        assert np.array_equal(A[k], B[k]), k
    assert torch.equal(JA, JB)
    moved = np.abs(A["uy"]).max() > 0 or np.abs(A["ux"]).max() > 0
    at_rest = ((A["ux"] == 0) & (A["uy"] == 0) & (A["uz"] == 0)).mean()
    assert moved and 0.2 < at_rest < 1.0, at_rest


@pytest.mark.parametrize("name", ["cfg1_tiny_cic", "cfg2_thermal_tsc_32", "cfg3_lwfa_tsc_32x128x32", "cfg5_pqs_32x32x16"])
def test_energy_conserving_gather_variant(name):
    """Option gather = 1 against the oracle's energy-conserving gather (pinned in
    tests/test_oracle_gather_ec.py): dense supercells through the one-phase kernel, sparse ones per particle."""
    import oracle
    wl, u_scale = CASES[name]
    parts, fields = W.make_particles(wl), W.make_fields(wl)
    if u_scale == "local":
        u_scale = PP.local_u_scale(wl, parts.x.numpy(), parts.y.numpy(), parts.z.numpy(), fields.numpy(), 2)
    orc = oracle.Oracle(wl.grid, wl.cell, wl.dt, wl.supercell, wl.shape_order, gather=1)
    orc.load_particles(*(getattr(parts, k).numpy() for k in ("x", "y", "z", "ux", "uy", "uz", "w")),
                       species=parts.species.numpy())
    orc.set_fields(fields.numpy())
    pic = PP.gpu_for(wl, parts, fields, gather=1)
    assert orc.step(2) == 0
    pic.step(2)
    pic.sync()
    rep = PP.compare(wl, orc, pic, 2, u_scale)
    print(f"\n[{name} gather=1] {rep}")
    assert rep.max_dx <= 2 * PP.TOL_X and rep.max_du_rel <= 2 * PP.TOL_U and rep.j_err_rel <= PP.TOL_J10
    assert rep.n_member_mismatch == 0 and rep.counts_equal_outside_band
    # and it is a different method: the momentum-conserving run differs by far more than the tolerance
    ref = PP.gpu_for(wl, parts, fields)
    ref.step(2)
    A, B = PP.gpu_particles_by_id(pic), PP.gpu_particles_by_id(ref)
    if name != "cfg1_tiny_cic":          # (uniform fields are gathered exactly by both)
        assert np.abs(A["ux"] - B["ux"]).max() > 1e-5 * float(np.abs(B["ux"]).max() + 1e-3)
    pic.destroy()
    ref.destroy()


@pytest.mark.parametrize("nosort", (0, 1, 4))
def test_all_sparse_steps_without_resort(nosort):
    """All-sparse workload (2 particles per cell, one thread per particle): with option sparse_nosort the steps run on
    the unsorted state (holes of leavers, appended arrivals) and sort once in 16 steps (option value 1) or in 4 (option
    value 4: the periodic sort inside a pic_step(n) call, several times).  20 free-running steps of a hot, sparse
    plasma (a few per cent of the particles change supercell per step, whole supercells of the slab boundary empty
    and fill) against the oracle, with and without the option; read-backs in between sort on demand."""
    wl = W.CONFIGS["lwfa"].scaled((32, 64, 16), u_th=0.25, ramp_cells=8)
    parts, fields = W.make_particles(wl), W.make_fields(wl) * 0.02
    orc = PP.oracle_for(wl, parts, fields)
    pic = PP.gpu_for(wl, parts, fields, sparse_nosort=nosort)
    for n in (3, 9, 8):
        assert orc.step(n) == 0
        pic.step(n)
        pic.sync()
        assert PP.gpu_membership_consistent(wl, pic)       # sorts the pending state for the read-back
    rep = PP.compare(wl, orc, pic, 20, 0.25)
    print(f"\n[all-sparse, sparse_nosort={nosort}] {rep} leavers={pic.get_stats()['leavers_cum']}")
    assert pic.get_stats()["error"] == 0 and pic.get_stats()["leavers_cum"] > parts.n // 4
    assert rep.max_dx <= 20 * PP.TOL_X and rep.max_du_rel <= 20 * PP.TOL_U and rep.j_err_rel <= PP.TOL_J10
    assert rep.n_member_mismatch == 0 and rep.counts_equal_outside_band
    pic.destroy()


@pytest.mark.parametrize("name", ["cfg1_tiny_cic", "cfg2_thermal_tsc_32", "cfg5_pqs_32x32x16"])
def test_float_atomic_deposit_variant(name):
    """Option deposit=0 (float atomics on the shared J tile) computes the same step."""
    rep, pic, wl = _run(name, 1, deposit=0)
    assert rep.max_dx <= PP.TOL_X and rep.max_du_rel <= PP.TOL_U and rep.j_err_rel <= PP.TOL_J1
    assert rep.n_member_mismatch == 0 and rep.counts_equal_outside_band
    pic.destroy()


def test_load_order_changes_J_only_by_rounding():
    """Two runs whose particles are loaded in different orders differ only by the fp32 rounding of the
    per-cell register sums (the shared tile and global J accumulate exactly, in fixed point)."""
    wl, _ = CASES["cfg2_thermal_tsc_32"]
    parts, fields = W.make_particles(wl), W.make_fields(wl)
    perm = torch.randperm(parts.n, generator=torch.Generator().manual_seed(5))
    shuffled = W.ParticleChunk(*(getattr(parts, k)[perm] for k in ("x", "y", "z", "ux", "uy", "uz", "w", "species")))
    Js = []
    for p in (parts, shuffled):
        pic = PP.gpu_for(wl, p, fields)
        pic.step(1)
        Js.append(pic.get_current().cpu().numpy().astype(np.float64))
        pic.destroy()
    scale = np.abs(Js[0]).max()
    assert scale > 0 and np.abs(Js[0] - Js[1]).max() <= 1e-6 * scale


@pytest.mark.parametrize("name", ["cfg1_tiny_cic", "cfg2_thermal_tsc_32", "cfg4_khi_hotspot_tsc_24", "cfg5_pqs_32x32x16"])
def test_ten_steps_free_running(name):
    rep, pic, wl = _run(name, 10)
    assert rep.max_dx <= 10 * PP.TOL_X
    assert rep.max_du_rel <= 10 * PP.TOL_U
    assert rep.j_err_rel <= PP.TOL_J10
    assert rep.n_member_mismatch == 0 and rep.counts_equal_outside_band
    pic.destroy()


@pytest.mark.parametrize("name", list(CASES))
def test_gpu_continuity(name):
    """The GPU's own J and positions satisfy the discrete continuity equation (S22)."""
    wl, _ = CASES[name]
    parts, fields = W.make_particles(wl), W.make_fields(wl)
    pic = PP.gpu_for(wl, parts, fields)
    pic.step(2)     # not from the pristine state: resorted frames, arrivals appended
    res = PP.gpu_continuity(wl, pic, [-1.0] * 16)
    print(f"\n[{name}] continuity residual {res:.3e}")
    assert res <= PP.TOL_CONT
    pic.destroy()


@pytest.mark.parametrize("name", ["cfg1_tiny_cic", "cfg2_thermal_tsc_32", "cfg4_khi_hotspot_tsc_24", "cfg5_pqs_32x32x16"])
def test_one_phase_variant(name):
    """Option two_phase=0 (gather per particle from the shared tile) computes the same step;
    the default is the two-phase path (per-cell stencils in registers), covered by every other test."""
    rep, pic, wl = _run(name, 1, two_phase=0)
    assert rep.max_dx <= PP.TOL_X and rep.max_du_rel <= PP.TOL_U and rep.j_err_rel <= PP.TOL_J1
    assert rep.n_member_mismatch == 0 and rep.counts_equal_outside_band
    pic.destroy()


@pytest.mark.parametrize("name", ["cfg2_thermal_tsc_32", "cfg3_lwfa_tsc_32x128x32", "cfg4_khi_hotspot_tsc_24"])
def test_unfused_sort_variant(name):
    """Option fuse_sort=0 (a separate sort kernel before every step instead of the sort in the step kernel's
    prologue) computes the same steps."""
    rep, pic, wl = _run(name, 3, fuse_sort=0)
    assert rep.max_dx <= 3 * PP.TOL_X and rep.max_du_rel <= 3 * PP.TOL_U and rep.j_err_rel <= PP.TOL_J10
    assert rep.n_member_mismatch == 0 and rep.counts_equal_outside_band
    pic.destroy()


def test_readbacks_between_steps_sort_the_pending_state():
    """A step leaves the supercells unsorted (the next step's kernel sorts them).  Read-backs in between must
    see — and leave behind — a consistent sorted state: five single steps with pic_get_counts / pic_get_particles
    after each give bit-identical particles to one call of five steps."""
    wl, _ = CASES["cfg2_thermal_tsc_32"]
    parts, fields = W.make_particles(wl), W.make_fields(wl)
    a = PP.gpu_for(wl, parts, fields)
    b = PP.gpu_for(wl, parts, fields)
    a.step(5)
    for i in range(5):
        b.step(1)
        counts = b.get_counts()
        assert int(counts.sum()) == parts.n
        if i % 2 == 0:
            assert b.get_particles()["id"].numel() == parts.n
    A, B = PP.gpu_particles_by_id(a), PP.gpu_particles_by_id(b)
    for k in ("x", "y", "z", "ux", "uy", "uz", "supercell"):
        assert np.array_equal(A[k], B[k]), k
    Ja, Jb = a.get_current().cpu().numpy(), b.get_current().cpu().numpy()
    assert np.abs(Ja - Jb).max() <= 1e-6 * np.abs(Ja).max()      # fp32 rounding of the per-item sums (order in a cell)
    assert torch.equal(a.get_counts(), b.get_counts())
    a.destroy(); b.destroy()


@pytest.mark.parametrize("cls", (0, 1, 2))
@pytest.mark.parametrize("name", ["cfg3_lwfa_tsc_32x128x32", "cfg4_khi_hotspot_tsc_24", "cfg5_pqs_32x32x16"])
def test_variant_choice_is_performance_only(name, cls):
    """Which step-kernel variants a step launches follows the host's (possibly stale) knowledge of the supercell
    populations; a supercell on the wrong side of the line is still stepped correctly by the variant that takes
    every supercell.  Forced here: everything through the sparse variant (1), through the dense ones (2),
    classified per supercell (0) — on workloads with sparse, dense and crowded supercells."""
    rep, pic, wl = _run(name, 3, class_all=cls)
    assert rep.max_dx <= 3 * PP.TOL_X and rep.max_du_rel <= 3 * PP.TOL_U and rep.j_err_rel <= PP.TOL_J10
    assert rep.n_member_mismatch == 0 and rep.counts_equal_outside_band
    pic.destroy()


@pytest.mark.parametrize("order,ppc", [(1, 40), (2, 33), (2, 40), (3, 18), (3, 30)])
def test_item_length_limits(order, ppc):
    """Cells that need several two-phase work items of maximal length (ppc well above the staging limit of
    11 / 6 particles per item), and supercells just below and above the population where the item list
    overflows and the one-phase variant takes over (768 x 11 = 8448 for CIC/TSC, 768 x 6 = 4608 for PQS)."""
    wl = W.CONFIGS["thermal_128"].scaled((16, 16, 8), shape_order=order, ppc=ppc)
    parts, fields = W.make_particles(wl), W.make_fields(wl)
    orc = PP.oracle_for(wl, parts, fields)
    pic = PP.gpu_for(wl, parts, fields)
    assert orc.step(2) == 0
    pic.step(2)
    rep = PP.compare(wl, orc, pic, 2, 0.05)
    print(f"\n[item limits order {order} ppc {ppc}] {rep}")
    assert rep.max_dx <= 2 * PP.TOL_X and rep.max_du_rel <= 2 * PP.TOL_U and rep.j_err_rel <= 2 * PP.TOL_J1
    assert rep.n_member_mismatch == 0 and rep.counts_equal_outside_band
    assert pic.get_stats()["error"] == 0
    pic.destroy()


@pytest.mark.parametrize("order", (1, 2, 3))
def test_fast_particles_leave_the_register_window(order):
    """c*dt = 0.9 cell and relativistic momenta: most particles move more than half a cell, leave their
    cell's 4-node register window, fill the shared-memory queue (768 per supercell) and spill into the
    on-the-spot deposit.  Same tolerances."""
    wl = W.CONFIGS["thermal_128"].scaled((16, 16, 8), shape_order=order, ppc=16, u_th=1.0, dt=0.9)
    parts, fields = W.make_particles(wl), W.make_fields(wl)
    orc = PP.oracle_for(wl, parts, fields)
    pic = PP.gpu_for(wl, parts, fields)
    assert orc.step(2) == 0
    pic.step(2)
    rep = PP.compare(wl, orc, pic, 2, 1.0)
    print(f"\n[fast particles order {order}] {rep}")
    assert rep.max_dx <= 2 * PP.TOL_X and rep.max_du_rel <= 2 * PP.TOL_U and rep.j_err_rel <= 2 * PP.TOL_J1
    assert rep.n_member_mismatch == 0 and rep.counts_equal_outside_band
    assert pic.get_stats()["error"] == 0
    pic.destroy()


def test_long_run_with_bunching_reuses_frames():
    """Static fields make the plasma bunch (max supercell population grows severalfold); supercells that
    shrink must return their frames, or the pool (sized for 9/8 of the particles) runs dry."""
    wl = W.CONFIGS["thermal_128"].scaled((32, 32, 32), amplitude=0.04)
    parts, fields = W.make_particles(wl), W.make_fields(wl)
    pic = PP.gpu_for(wl, parts, fields)
    first = None
    for _ in range(6):
        pic.step(25)
        st = pic.get_stats()
        assert st["error"] == 0 and st["particles"] == parts.n
        first = first or st
    assert st["max_count"] > 1.5 * 4096, (first, st)      # the densest supercell grew well beyond the mean
    assert st["frames_used"] <= st["frames_pool"]
    assert PP.gpu_membership_consistent(wl, pic)
    assert int(pic.get_counts().sum()) == parts.n
    ids = pic.get_particles()["id"].to(torch.int64) & 0xFFFFFFFF
    assert torch.equal(torch.sort(ids).values, torch.arange(parts.n, device=ids.device))
    res = PP.gpu_continuity(wl, pic, [-1.0] * 16)
    print(f"\n[long run] max_count {first['max_count']} -> {st['max_count']}, frames {st['frames_used']}/{st['frames_pool']}, continuity {res:.2e}")
    assert res <= PP.TOL_CONT
    pic.destroy()


def test_species_table_and_anisotropic_cells():
    """Positive charge / heavier species and dx != dy != dz go through the same kernels."""
    wl = W.CONFIGS["khi"].scaled((16, 24, 8), cell=(1.0, 0.8, 1.25), dt=0.4)
    parts, fields = W.make_particles(wl), W.make_fields(wl)
    orc = PP.oracle_for(wl, parts, fields)
    orc.set_species([-1.0, 2.0], [1.0, 4.0])
    pic = PP.gpu_for(wl, parts, fields)
    pic.set_species([-1.0, 2.0], [1.0, 4.0])
    assert orc.step(3) == 0
    pic.step(3)
    rep = PP.compare(wl, orc, pic, 3, 0.01)
    print(f"\n[species/anisotropic] {rep}")
    assert rep.max_dx <= 3 * PP.TOL_X and rep.max_du_rel <= 3 * PP.TOL_U and rep.j_err_rel <= 3 * PP.TOL_J1
    assert rep.n_member_mismatch == 0
    pic.destroy()


def test_append_loads_and_empty_supercells():
    """Repeated pic_load_particles calls append; supercells without particles are fine."""
    wl = W.CONFIGS["lwfa"].scaled((16, 64, 8))
    fields = W.make_fields(wl)
    chunks = list(W.particle_chunks(wl, max_chunk=2048))
    assert len(chunks) > 2
    parts = W.ParticleChunk.cat(chunks)
    orc = PP.oracle_for(wl, parts, fields)
    from paper_2110_08650_b200.binding import Pic
    pic = Pic(wl.grid, wl.cell, wl.dt, wl.supercell, wl.shape_order, max_particles=parts.n)
    for c in chunks:
        g = c.to("cuda:0")
        pic.load_particles(g.x, g.y, g.z, g.ux, g.uy, g.uz, g.w, g.species)
        pic.sync()
    pic.set_fields(fields.cuda())
    counts0 = pic.get_counts().cpu().numpy()
    assert counts0.sum() == parts.n and (counts0 == 0).any()
    assert orc.step(2) == 0
    pic.step(2)
    rep = PP.compare(wl, orc, pic, 2, 0.5)
    print(f"\n[append] {rep}")
    assert rep.max_dx <= 2 * PP.TOL_X and rep.max_du_rel <= 2 * PP.TOL_U and rep.j_err_rel <= 2 * PP.TOL_J1
    assert rep.n_member_mismatch == 0
    pic.destroy()


def test_load_more_particles_between_steps():
    """pic_load_particles after stepping appends to the cell-sorted state (ids continue)."""
    wl = W.CONFIGS["khi"].scaled((16, 16, 16))
    parts, fields = W.make_particles(wl), W.make_fields(wl)
    keys = ("x", "y", "z", "ux", "uy", "uz", "w", "species")
    perm = torch.randperm(parts.n, generator=torch.Generator().manual_seed(3))
    half = [W.ParticleChunk(*(getattr(parts, k)[idx] for k in keys)) for idx in (perm[: parts.n // 2], perm[parts.n // 2:])]
    from paper_2110_08650_b200.binding import Pic
    import oracle
    pic = Pic(wl.grid, wl.cell, wl.dt, wl.supercell, wl.shape_order, max_particles=parts.n)
    orc = oracle.Oracle(wl.grid, wl.cell, wl.dt, wl.supercell, wl.shape_order)
    pic.set_fields(fields.cuda())
    orc.set_fields(fields.numpy())
    for h in half:
        g = h.to("cuda:0")
        pic.load_particles(*(getattr(g, k) for k in keys))
        orc.load_particles(*(getattr(h, k).numpy() for k in keys[:7]), species=h.species.numpy())
        pic.step(2)
        assert orc.step(2) == 0
    rep = PP.compare(wl, orc, pic, 4, 0.01)
    print(f"\n[load between steps] {rep}")
    assert rep.max_dx <= 4 * PP.TOL_X and rep.max_du_rel <= 4 * PP.TOL_U and rep.j_err_rel <= 4 * PP.TOL_J1
    assert rep.n_member_mismatch == 0
    pic.destroy()


def test_roundtrip_without_step():
    """load -> get returns the same multiset, exactly (positions are integer + fp32 fraction)."""
    wl = W.CONFIGS["thermal_128"].scaled((16, 16, 8), ppc=5)
    parts = W.make_particles(wl)
    pic = PP.gpu_for(wl, parts, W.make_fields(wl))
    G = PP.gpu_particles_by_id(pic)
    for k in ("x", "y", "z", "ux", "uy", "uz", "w", "species"):
        assert np.array_equal(G[k], getattr(parts, k).numpy()), k
    assert PP.gpu_membership_consistent(wl, pic)
    pic.destroy()


def test_error_paths():
    from paper_2110_08650_b200.binding import Pic, PicError, PIC_EINVAL, PIC_ESTATE, PIC_ENOMEM
    with pytest.raises(PicError) as e:
        Pic((20, 16, 16), max_particles=10)            # not a multiple of the supercell
    assert e.value.code == PIC_EINVAL
    with pytest.raises(PicError) as e:
        Pic((16, 16, 16), dt=1.5, max_particles=10)    # c*dt >= cell
    assert e.value.code == PIC_EINVAL
    pic = Pic((16, 16, 16), max_particles=4)
    with pytest.raises(PicError) as e:
        pic.step(1)                                    # no fields yet
    assert e.value.code == PIC_ESTATE
    z64 = torch.zeros(8, dtype=torch.float64, device="cuda")
    z32 = torch.zeros(8, dtype=torch.float32, device="cuda")
    with pytest.raises(PicError) as e:
        pic.load_particles(z64, z64, z64, z32, z32, z32, z32)   # over capacity
    assert e.value.code == PIC_ENOMEM
    pic.destroy()
