"""-m gpu parity tests: the CUDA path (through the C-ABI binding) against the fp64 oracle on the same seeded
inputs.  Bars (BASELINE.json): neighbour lists exactly as sets; |dE|/|E| <= 1e-5; max |dF| <= 1e-3."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import nnp_oracle as orc          # noqa: E402
from paper_2405_01491_b200 import inputs, nnp  # noqa: E402
from tests import gpu_util as U               # noqa: E402


@pytest.fixture(scope="module")
def model1():
    return U.make_model(1)


def _rlist(rc, skin):
    return float(np.float32(rc) + np.float32(skin))


def _check_lists(ctx, xyz, box, n, skin, mol_id=None, method="brute"):
    for which, rc in ((0, 5.1), (1, 3.5)):
        got = U.gpu_neighbors(ctx, which, n)
        ref = orc.neighbors(xyz, box, _rlist(rc, skin), mol_id=mol_id, fp32_pred=True, method=method)
        bad = [i for i in range(n) if not np.array_equal(got[i], ref[i])]
        assert not bad, (which, len(bad), bad[:5])


# ---------------------------------------------------------------- config 1: 64 waters, tiny box (2 cells / side)
def test_config1_water64(model1):
    consts, widths, params, om = model1
    sp, xyz, box = inputs.water_box(64, 12.42)
    ctx = U.gpu_create(consts, widths, params, 1, len(sp))
    try:
        Eg, Fg = U.gpu_energy_forces(ctx, sp, xyz, box)
        _check_lists(ctx, xyz, box, len(sp), 0.0)
        ref = orc.energy_forces(om, sp, xyz, box)
        U.assert_parity(Eg, Fg, ref)
        # AEV hook, element by element
        d_aev = torch.zeros((len(sp), 1008), dtype=torch.float32, device="cuda")
        nnp.nnp_get_aev(ctx, d_aev)
        nnp.nnp_sync(ctx)
        aev_ref = orc.energy_forces(om, sp, xyz, box, want_forces=False, want_aev=True)["aev"]
        assert np.abs(d_aev.cpu().numpy() - aev_ref).max() < 2e-5 * max(1.0, np.abs(aev_ref).max())
        # with a skin: same energies and forces from the longer lists (reading A4)
        Eg2, Fg2 = U.gpu_energy_forces(ctx, sp, xyz, box, skin=0.5)
        _check_lists(ctx, xyz, box, len(sp), 0.5)
        U.assert_parity(Eg2, Fg2, ref)
    finally:
        nnp.nnp_destroy(ctx)


def test_unwrapped_coordinates_and_box_error(model1):
    consts, widths, params, om = model1
    sp, xyz, box = inputs.water_box(64, 12.42, seed=7)
    xyz = (xyz + np.random.default_rng(0).integers(-3, 4, size=xyz.shape) * box).astype(np.float32).astype(np.float64)
    ctx = U.gpu_create(consts, widths, params, 1, len(sp))
    try:
        Eg, Fg = U.gpu_energy_forces(ctx, sp, xyz, box)
        _check_lists(ctx, xyz, box, len(sp), 0.0)
        U.assert_parity(Eg, Fg, orc.energy_forces(om, sp, xyz, box))
        with pytest.raises(nnp.NnpError) as e:      # 12.42 < 2*(5.1+1.2)
            U.gpu_energy_forces(ctx, sp, xyz, box, skin=1.2)
        assert e.value.status == nnp.NNP_EBOX
    finally:
        nnp.nnp_destroy(ctx)


# ---------------------------------------------------------------- medium water box: several cells, ragged GEMM tiles
def test_water_1000_cells_and_tails(model1):
    consts, widths, params, om = model1
    sp, xyz, box = inputs.water_box(1000, seed=3)           # 3000 atoms, L = 31.04 A -> 6 cells / side at 5.1 A
    ctx = U.gpu_create(consts, widths, params, 1, len(sp))
    try:
        Eg, Fg = U.gpu_energy_forces(ctx, sp, xyz, box)
        _check_lists(ctx, xyz, box, len(sp), 0.0, method="grid")
        U.assert_parity(Eg, Fg, orc.energy_forces(om, sp, xyz, box, nbr_method=1))
    finally:
        nnp.nnp_destroy(ctx)


# ---------------------------------------------------------------- config 2 shape: 8-net ensemble (reduced size)
def test_ensemble_8_nets_water():
    consts, widths, params, om = U.make_model(8, seed=inputs.SEED0 + 2)
    sp, xyz, box = inputs.water_box(343, seed=4)
    ctx = U.gpu_create(consts, widths, params, 8, len(sp))
    try:
        Eg, Fg = U.gpu_energy_forces(ctx, sp, xyz, box)
        U.assert_parity(Eg, Fg, orc.energy_forces(om, sp, xyz, box, nbr_method=1))
    finally:
        nnp.nnp_destroy(ctx)


# ---------------------------------------------------------------- config 4 shape: all 7 species, uneven buckets
def test_mixed_species_solvated_chain(model1):
    consts, widths, params, om = model1
    sp, xyz, box = inputs.solvated_chain(n_solute=600, L=24.0, seed=5)
    sp = sp.copy()
    sp[:14] = np.arange(14) % 7          # every species present even in this reduced system
    assert len(np.unique(sp)) == 7
    ctx = U.gpu_create(consts, widths, params, 1, len(sp))
    try:
        Eg, Fg = U.gpu_energy_forces(ctx, sp, xyz, box)
        _check_lists(ctx, xyz, box, len(sp), 0.0, method="grid")
        U.assert_parity(Eg, Fg, orc.energy_forces(om, sp, xyz, box, nbr_method=1))
    finally:
        nnp.nnp_destroy(ctx)


# ---------------------------------------------------------------- config 5 shape: batched non-periodic molecules
def test_molecule_batch(model1):
    consts, widths, params, om = U.make_model(2, seed=inputs.SEED0 + 5)
    sp, xyz, offs = inputs.molecule_batch(300, seed=12)
    mol = np.repeat(np.arange(300), np.diff(offs)).astype(np.int32)
    ctx = U.gpu_create(consts, widths, params, 2, len(sp), max_mols=300)
    try:
        Eg, Fg = U.gpu_energy_forces(ctx, sp, xyz, None, mol_offsets=offs)
        _check_lists(ctx, xyz, None, len(sp), 0.0, mol_id=mol)
        ref = orc.energy_forces(om, sp, xyz, None, offs, want_e_atom=True)
        U.assert_parity(Eg, Fg, ref, mol_offsets=offs)
        # the plain 1e-5 relative bar holds for every structure whose atomic energies do not cancel
        big = np.abs(ref["E"]) > 0.5 * np.array([np.abs(ref["e_atom"][offs[m]:offs[m + 1]]).sum() for m in range(300)])
        assert big.sum() > 30
        assert (np.abs(Eg - ref["E"])[big] <= U.E_RTOL * np.abs(ref["E"])[big]).all()
    finally:
        nnp.nnp_destroy(ctx)


# ---------------------------------------------------------------- replicas of one periodic cell in one batch
@pytest.mark.parametrize("n_waters, L, n_rep", [(64, 12.42, 5), (1000, None, 3)], ids=["tiny_box_x5", "water1000_x3"])
def test_periodic_replica_batch(model1, n_waters, L, n_rep):
    """RPMD-style replica batching: n_rep perturbed copies of one periodic water box in one call; lists
    exactly those of the oracle (never across replicas), per-replica energies and all forces against the oracle."""
    consts, widths, params, om = model1
    sp1, x1, box = inputs.water_box(n_waters, L, seed=inputs.SEED0 + 9)
    rng = np.random.default_rng(5)
    reps = [(x1 + 0.04 * rng.standard_normal(x1.shape) * (r > 0)).astype(np.float32).astype(np.float64) for r in range(n_rep)]
    sp = np.tile(sp1, n_rep)
    xyz = np.concatenate(reps)
    offs = (np.arange(n_rep + 1) * len(sp1)).astype(np.int32)
    mol = np.repeat(np.arange(n_rep), len(sp1)).astype(np.int32)
    ctx = U.gpu_create(consts, widths, params, 1, len(sp), max_mols=n_rep)
    try:
        Eg, Fg = U.gpu_energy_forces(ctx, sp, xyz, box, mol_offsets=offs)
        _check_lists(ctx, xyz, box, len(sp), 0.0, mol_id=mol)
        ref = orc.energy_forces(om, sp, xyz, box, offs, want_e_atom=True)
        U.assert_parity(Eg, Fg, ref, mol_offsets=offs)
        assert (np.abs(Eg - ref["E"]) <= U.E_RTOL * np.abs(ref["E"])).all()
        # with a skin, and the same replicas one at a time through the single-structure path
        Es, Fs = U.gpu_energy_forces(ctx, sp, xyz, box, mol_offsets=offs, skin=0.4)
        U.assert_parity(Es, Fs, ref, mol_offsets=offs)
        E1, F1 = U.gpu_energy_forces(ctx, sp1, reps[1], box)
        assert abs(E1[0] - Eg[1]) <= 2e-6 * abs(Eg[1]) and np.abs(F1 - Fg[offs[1]:offs[2]]).max() < 2e-4
    finally:
        nnp.nnp_destroy(ctx)


# ---------------------------------------------------------------- the other matmul modes on an ensemble
@pytest.mark.parametrize("mm_mode", [nnp.NNP_MM_FP32_SIMT, nnp.NNP_MM_3XTF32_TC, nnp.NNP_MM_3XF16_TC], ids=["fp32_simt", "3xtf32_tc", "3xf16_fused"])
def test_ensemble_in_both_fp32_grade_modes(mm_mode):
    """Three networks on a 216-water box: the fp32 SIMT path runs the networks one after the other, the 3xTF32 path batches
    them into one grouped launch per layer, the fused 3xF16 chain takes all of them in one launch (dE/dG summed by
    reductions in memory in both tensor-core paths); all meet the bars."""
    consts, widths, params, om = U.make_model(3, seed=inputs.SEED0 + 21)
    sp, xyz, box = inputs.water_box(216, seed=inputs.SEED0 + 22)
    ctx = U.gpu_create(consts, widths, params, 3, len(sp), mm_mode=mm_mode)
    try:
        Eg, Fg = U.gpu_energy_forces(ctx, sp, xyz, box)
        ref = orc.energy_forces(om, sp, xyz, box, want_e_atom=True)
        U.assert_parity(Eg, Fg, ref)                                  # reading B8: E is a cancelling sum here ...
        U.assert_strict_energy_bar_where_it_is_defined(Eg, ref)      # ... and the strict bar applies if it is not
    finally:
        nnp.nnp_destroy(ctx)


@pytest.mark.parametrize("mm_mode", [nnp.NNP_MM_3XTF32_TC, nnp.NNP_MM_3XF16_TC], ids=["3xtf32_six_launches", "3xf16_fused"])
def test_both_tensor_core_modes_on_every_chain(mm_mode):
    """The suite runs in ONE matmul mode (NNP_MM_MODE, default 4); this test takes the other fp32-grade tensor-core mode
    through the same shapes: water (128 active AEV columns, row tiles with a ragged tail), all seven species (1024 columns: the
    fused chain streams its first and last GEMM in passes; buckets from 2 to ~1000 rows) and a molecule batch with two networks."""
    consts, widths, params, om = U.make_model(1)
    sp, xyz, box = inputs.water_box(1000, seed=3)
    ctx = U.gpu_create(consts, widths, params, 1, 3600, mm_mode=mm_mode)
    try:
        Eg, Fg = U.gpu_energy_forces(ctx, sp, xyz, box)
        U.assert_parity(Eg, Fg, orc.energy_forces(om, sp, xyz, box, nbr_method=1))
        sp, xyz, box = inputs.solvated_chain(n_solute=600, L=24.0, seed=5)
        sp = sp.copy()
        sp[:14] = np.arange(14) % 7
        Eg, Fg = U.gpu_energy_forces(ctx, sp, xyz, box)
        U.assert_parity(Eg, Fg, orc.energy_forces(om, sp, xyz, box, nbr_method=1))
    finally:
        nnp.nnp_destroy(ctx)
    consts, widths, params, om = U.make_model(2, seed=inputs.SEED0 + 5)
    sp, xyz, offs = inputs.molecule_batch(120, seed=12)
    ctx = U.gpu_create(consts, widths, params, 2, len(sp), max_mols=120, mm_mode=mm_mode)
    try:
        Eg, Fg = U.gpu_energy_forces(ctx, sp, xyz, None, mol_offsets=offs)
        U.assert_parity(Eg, Fg, orc.energy_forces(om, sp, xyz, None, offs, want_e_atom=True), mol_offsets=offs)
    finally:
        nnp.nnp_destroy(ctx)


def test_fused_mode_reports_activations_out_of_fp16_range():
    """mm_mode 4 scales activations by 16 into fp16 hi/lo operands: |value| > 3750 must come back as NNP_ERANGE, never as
    a silently saturated energy.  A last layer 1e4 times the parity tests' makes delta3 = w4 celu'(h3) that large."""
    consts, widths, params, om = U.make_model(1, scale=U.FORCE_SCALE * 1e4)
    sp, xyz, box = inputs.water_box(64, 12.42)
    ctx = U.gpu_create(consts, widths, params, 1, len(sp), mm_mode=nnp.NNP_MM_3XF16_TC)
    try:
        with pytest.raises(nnp.NnpError) as ei:
            U.gpu_energy_forces(ctx, sp, xyz, box)
        assert ei.value.status == nnp.NNP_ERANGE
    finally:
        nnp.nnp_destroy(ctx)
    # the same model through 3xTF32 (tf32 carries the fp32 exponent) evaluates fine
    ctx = U.gpu_create(consts, widths, params, 1, len(sp), mm_mode=nnp.NNP_MM_3XTF32_TC)
    try:
        Eg, Fg = U.gpu_energy_forces(ctx, sp, xyz, box)
        ref = orc.energy_forces(om, sp, xyz, box)
        assert abs(Eg[0] - ref["E"][0]) <= U.E_RTOL * abs(ref["E"][0])
    finally:
        nnp.nnp_destroy(ctx)


# ---------------------------------------------------------------- degenerate inputs
def test_edge_cases(model1):
    consts, widths, params, om = model1
    ctx = U.gpu_create(consts, widths, params, 1, 64, max_mols=4)
    try:
        # empty system
        Eg, Fg = U.gpu_energy_forces(ctx, np.zeros(0, np.int32), np.zeros((0, 3)), None)
        assert Eg[0] == 0.0
        # single isolated atom: energy = network(0) = bias chain
        Eg, Fg = U.gpu_energy_forces(ctx, [3], [[0.0, 0.0, 0.0]], None)
        ref = orc.energy_forces(om, [3], [[0.0, 0.0, 0.0]])
        assert abs(Eg[0] - ref["E"][0]) <= 1e-5 * abs(ref["E"][0]) and np.all(Fg == 0)
        # dimer and collinear trimer
        for sp, xyz in (([0, 0], [[0, 0, 0], [0.74, 0, 0]]), ([3, 0, 0], [[0, 0, 0], [0.96, 0, 0], [-0.96, 0, 0]])):
            Eg, Fg = U.gpu_energy_forces(ctx, sp, xyz, None)
            U.assert_parity(Eg, Fg, orc.energy_forces(om, sp, xyz))
        # batch containing 1-atom molecules
        sp = [0, 3, 0, 0, 1]
        xyz = [[0, 0, 0], [5, 5, 5], [5.9, 5, 5], [5, 5.9, 5], [9, 9, 9]]
        offs = [0, 1, 4, 5]
        Eg, Fg = U.gpu_energy_forces(ctx, sp, xyz, None, mol_offsets=offs)
        U.assert_parity(Eg, Fg, orc.energy_forces(om, sp, xyz, None, offs))
        # bad species index is rejected
        with pytest.raises(nnp.NnpError):
            U.gpu_energy_forces(ctx, [9], [[0, 0, 0]], None)
        # energy_forces without lists
        d = torch.zeros((1, 3), device="cuda")
        nnp.nnp_set_system(ctx, 1, torch.zeros(1, dtype=torch.int32, device="cuda"), d, None)
        with pytest.raises(nnp.NnpError) as e:
            nnp.nnp_energy_forces(ctx, torch.zeros(1, dtype=torch.float64, device="cuda"), d)
        assert e.value.status == nnp.NNP_ESTALE
    finally:
        nnp.nnp_destroy(ctx)


def test_capacity_overflow_is_reported(model1):
    consts, widths, params, om = model1
    sp, xyz, box = inputs.water_box(64, 12.42)
    ctx = U.gpu_create(consts, widths, params, 1, len(sp), cap_r=32, cap_a=64)
    try:
        with pytest.raises(nnp.NnpError) as e:
            U.gpu_energy_forces(ctx, sp, xyz, box)
        assert e.value.status == nnp.NNP_ECAPACITY
    finally:
        nnp.nnp_destroy(ctx)


# ---------------------------------------------------------------- MD (stage 5)
@pytest.mark.parametrize("graph", [False, True], ids=["kernel_by_kernel", "cuda_graph"])
def test_md_steps_against_oracle(model1, graph):
    """graph=True: the context runs on a side stream, so nnp_md_step launches the captured step graph (rebuild inside
    a conditional node); graph=False: default stream, every kernel enqueued separately."""
    consts, widths, params, om = model1
    sp, xyz, box = inputs.water_box(216, seed=9)
    v = inputs.maxwell_boltzmann(sp, 300.0, seed=2)
    n = len(sp)
    dev = torch.device("cuda:0")
    ctx = U.gpu_create(consts, widths, params, 1, n, stream=torch.cuda.Stream(device=dev) if graph else None)
    try:
        d_sp = torch.as_tensor(sp, device=dev)
        d_x = torch.as_tensor(xyz.astype(np.float32), device=dev)
        d_v = torch.as_tensor(v.astype(np.float32), device=dev)
        torch.cuda.synchronize()
        nnp.nnp_set_system(ctx, n, d_sp, d_x, box)
        nnp.nnp_md_init(ctx, d_v, 0.5, 0.5)
        o_x, o_v = torch.zeros_like(d_x), torch.zeros_like(d_v)
        o_ep = torch.zeros(1, dtype=torch.float64, device=dev)
        o_ek = torch.zeros(1, dtype=torch.float64, device=dev)
        o_nr = torch.zeros(1, dtype=torch.int32, device=dev)
        torch.cuda.synchronize()

        def state():
            nnp.nnp_get_state(ctx, o_x, o_v, o_ep, o_ek, o_nr)
            nnp.nnp_sync(ctx)
            return (o_x.cpu().numpy().astype(np.float64), o_v.cpu().numpy().astype(np.float64),
                    float(o_ep.item()), float(o_ek.item()), int(o_nr.item()))

        x0, v0, ep0, ek0, nr0 = state()
        assert nr0 == 1 and np.array_equal(x0, xyz) and np.array_equal(v0, v)
        ref0 = orc.energy_forces(om, sp, xyz, box)
        assert abs(ep0 - ref0["E"][0]) <= U.E_RTOL * abs(ref0["E"][0])
        ke0 = 0.5 * (inputs.MASS[sp][:, None] * v ** 2).sum() / inputs.ACCEL_CONV
        assert abs(ek0 - ke0) <= 1e-5 * ke0

        # one step against the oracle integrator started from the same state
        nnp.nnp_md_step(ctx, 1)
        x1, v1, ep1, ek1, nr1 = state()
        o1 = orc.md(om, sp, xyz, v, inputs.MASS, box, 0.5, inputs.ACCEL_CONV, 1)
        assert np.abs(x1 - o1["xyz"]).max() < 2e-6 and np.abs(v1 - o1["vel"]).max() < 2e-6
        assert abs(ep1 - o1["epot"][1]) <= 2e-5 * abs(o1["epot"][1])

        # 60 more steps: the lists must have been rebuilt by the displacement rule and must still be valid:
        # E and F of the GPU state, recomputed by the oracle at the GPU's positions, agree
        tot = [ep1 + ek1]
        for _ in range(6):
            nnp.nnp_md_step(ctx, 10)
            xs, vs, ep, ek, nr = state()
            tot.append(ep + ek)
        assert nr >= 3
        ref = orc.energy_forces(om, sp, xs, box)
        assert abs(ep - ref["E"][0]) <= U.E_RTOL * abs(ref["E"][0])
        # forces at the final state through a fresh evaluation of the same positions
        Eg, Fg = U.gpu_energy_forces(ctx, sp, xs, box, skin=0.5)
        U.assert_parity(Eg, Fg, ref)
        # NVE: total energy conserved to integrator accuracy (< 0.1 % criterion)
        tot = np.array(tot)
        assert np.abs(tot - tot[0]).max() < 1e-3 * abs(ek0) + 1e-3 * abs(tot[0])
    finally:
        nnp.nnp_destroy(ctx)


@pytest.mark.parametrize("graph", [False, True], ids=["kernel_by_kernel", "cuda_graph"])
def test_md_on_a_replica_batch(model1, graph):
    """SURVEY 8(f)-4 / PAPER.md L309: the replicas of a ring polymer take their MD steps as ONE batch.  Four replicas of a
    125-water cell (different positions and velocities) step together; each must follow the oracle's integrator run on that
    replica alone, energies come back per replica, and after 40 steps (lists rebuilt by the shared displacement flag) the
    oracle's E and F at the GPU's positions agree replica by replica."""
    consts, widths, params, om = model1
    n_rep = 4
    sp1, x1, box = inputs.water_box(125, seed=inputs.SEED0 + 31)
    n1 = len(sp1)
    rng = np.random.default_rng(11)
    reps = [(x1 + 0.03 * rng.standard_normal(x1.shape) * (r > 0)).astype(np.float32).astype(np.float64) for r in range(n_rep)]
    vels = [inputs.maxwell_boltzmann(sp1, 300.0, seed=40 + r).astype(np.float32).astype(np.float64) for r in range(n_rep)]
    sp, xyz, v = np.tile(sp1, n_rep), np.concatenate(reps), np.concatenate(vels)
    offs = (np.arange(n_rep + 1) * n1).astype(np.int32)
    n = len(sp)
    dev = torch.device("cuda:0")
    ctx = U.gpu_create(consts, widths, params, 1, n, max_mols=n_rep, stream=torch.cuda.Stream(device=dev) if graph else None)
    try:
        d_sp = torch.as_tensor(sp.astype(np.int32), device=dev)
        d_x = torch.as_tensor(xyz.astype(np.float32), device=dev)
        d_v = torch.as_tensor(v.astype(np.float32), device=dev)
        d_o = torch.as_tensor(offs, device=dev)
        torch.cuda.synchronize()
        nnp.nnp_set_system(ctx, n, d_sp, d_x, box, n_rep, d_o)
        nnp.nnp_md_init(ctx, d_v, 0.5, 0.5)
        o_x, o_v = torch.zeros_like(d_x), torch.zeros_like(d_v)
        o_ep = torch.zeros(n_rep, dtype=torch.float64, device=dev)
        o_ek = torch.zeros(n_rep, dtype=torch.float64, device=dev)
        o_nr = torch.zeros(1, dtype=torch.int32, device=dev)
        torch.cuda.synchronize()

        def state():
            nnp.nnp_get_state(ctx, o_x, o_v, o_ep, o_ek, o_nr)
            nnp.nnp_sync(ctx)
            return (o_x.cpu().numpy().astype(np.float64), o_v.cpu().numpy().astype(np.float64),
                    o_ep.cpu().numpy(), o_ek.cpu().numpy(), int(o_nr.item()))

        x0, v0, ep0, ek0, nr0 = state()
        for r in range(n_rep):
            ke = 0.5 * (inputs.MASS[sp1][:, None] * vels[r] ** 2).sum() / inputs.ACCEL_CONV
            assert abs(ek0[r] - ke) <= 1e-5 * ke
        nnp.nnp_md_step(ctx, 2)
        x2, v2, ep2, ek2, nr2 = state()
        for r in range(n_rep):
            o = orc.md(om, sp1, reps[r], vels[r], inputs.MASS, box, 0.5, inputs.ACCEL_CONV, 2)
            sl = slice(offs[r], offs[r + 1])
            assert np.abs(x2[sl] - o["xyz"]).max() < 4e-6 and np.abs(v2[sl] - o["vel"]).max() < 4e-6, r
            assert abs(ep2[r] - o["epot"][2]) <= 2e-5 * abs(o["epot"][2]) and abs(ek2[r] - o["ekin"][2]) <= 1e-4 * o["ekin"][2], r
        tot0 = ep2 + ek2
        nnp.nnp_md_step(ctx, 38)
        xs, vs, ep, ek, nr = state()
        assert nr >= 2
        tot = ep + ek
        for r in range(n_rep):
            sl = slice(offs[r], offs[r + 1])
            ref = orc.energy_forces(om, sp1, xs[sl], box)
            assert abs(ep[r] - ref["E"][0]) <= U.E_RTOL * abs(ref["E"][0]), r
            assert abs(tot[r] - tot0[r]) < 1e-3 * abs(ek2[r]) + 1e-3 * abs(tot0[r]), r     # every replica conserves its own energy
        # the host entry point returns the scalars of one structure only
        h = np.zeros((n, 3), dtype=np.float32)
        with pytest.raises(nnp.NnpError) as e:
            nnp.nnp_md_step_host(ctx, h, h.copy(), 1, np.zeros(1), np.zeros(1))
        assert e.value.status == nnp.NNP_EINVAL
    finally:
        nnp.nnp_destroy(ctx)


def test_host_entry_points_roundtrip(model1):
    consts, widths, params, om = model1
    sp, xyz, box = inputs.water_box(125, seed=10)
    n = len(sp)
    ctx = U.gpu_create(consts, widths, params, 1, n)
    try:
        h_sp = np.ascontiguousarray(sp, dtype=np.int32)
        h_x = np.ascontiguousarray(xyz, dtype=np.float32)
        h_E = np.zeros(1)
        h_F = np.zeros((n, 3), dtype=np.float32)
        nnp.nnp_energy_forces_host(ctx, n, h_sp, h_x, box, 1, None, 0.0, h_E, h_F)
        ref = orc.energy_forces(om, sp, xyz, box)
        U.assert_parity(h_E, h_F.astype(np.float64), ref)
        # MD through host buffers equals MD through device buffers
        v = inputs.maxwell_boltzmann(sp, 300.0, seed=3).astype(np.float32)
        dev = torch.device("cuda:0")
        nnp.nnp_set_system(ctx, n, torch.as_tensor(h_sp, device=dev), torch.as_tensor(h_x, device=dev), box)
        nnp.nnp_md_init(ctx, torch.as_tensor(v, device=dev), 0.5, 0.5)
        hx, hv = h_x.copy(), v.copy()
        ep, ek = np.zeros(1), np.zeros(1)
        for _ in range(5):
            nnp.nnp_md_step_host(ctx, hx, hv, 1, ep, ek)
        o = orc.md(om, sp, xyz, v.astype(np.float64), inputs.MASS, box, 0.5, inputs.ACCEL_CONV, 5)
        assert np.abs(hx - o["xyz"]).max() < 1e-5 and np.abs(hv - o["vel"]).max() < 1e-5
        assert abs(ep[0] - o["epot"][5]) <= 5e-5 * abs(o["epot"][5])
    finally:
        nnp.nnp_destroy(ctx)


# ---------------------------------------------------------------- BASELINE.json's full sizes, in the launch
# configuration bench.py times (persistent AEV kernels, tcgen05 grouped GEMMs over full buckets).  The oracle
# evaluates the same inputs in full (its grid neighbour search); neighbour rows are compared on a sample.
def _sampled_lists(ctx, xyz, box, n, skin, mol_id=None, n_sample=2000, seed=0):
    pick = np.random.default_rng(seed).choice(n, size=min(n, n_sample), replace=False)
    for which, rc in ((0, 5.1), (1, 3.5)):
        got = U.gpu_neighbors(ctx, which, n)
        ref = orc.neighbors(xyz, box, _rlist(rc, skin), mol_id=mol_id, fp32_pred=True,
                            method="grid" if box is not None else "brute")
        bad = [int(i) for i in pick if not np.array_equal(got[i], ref[i])]
        assert not bad, (which, len(bad), bad[:5])
        assert sum(len(r) for r in got) == sum(len(r) for r in ref)     # every row, by count


def test_full_config2_water12288_ensemble8():
    consts, widths, params, om = U.make_model(8, seed=inputs.SEED0 + 2)
    sp, xyz, box = inputs.water_box(4096, 49.7, seed=inputs.SEED0 + 2)
    assert len(sp) == 12288
    ctx = U.gpu_create(consts, widths, params, 8, len(sp))
    try:
        Eg, Fg = U.gpu_energy_forces(ctx, sp, xyz, box)
        _sampled_lists(ctx, xyz, box, len(sp), 0.0)
        U.assert_parity(Eg, Fg, orc.energy_forces(om, sp, xyz, box, nbr_method=1))
    finally:
        nnp.nnp_destroy(ctx)


def test_full_config3_water98304_md(model1):
    consts, widths, params, om = model1
    sp, xyz, box = inputs.water_box(32768, 99.4, seed=inputs.SEED0 + 3)
    n = len(sp)
    assert n == 98304
    v = inputs.maxwell_boltzmann(sp, 300.0, seed=inputs.SEED0 + 103)
    dev = torch.device("cuda:0")
    ctx = U.gpu_create(consts, widths, params, 1, n)
    try:
        nnp.nnp_set_system(ctx, n, torch.as_tensor(sp, device=dev), torch.as_tensor(xyz.astype(np.float32), device=dev), box)
        nnp.nnp_md_init(ctx, torch.as_tensor(v.astype(np.float32), device=dev), 0.5, 0.5)
        _sampled_lists(ctx, xyz, box, n, 0.5)
        nnp.nnp_md_step(ctx, 25)
        o_x = torch.zeros((n, 3), dtype=torch.float32, device=dev)
        o_ep = torch.zeros(1, dtype=torch.float64, device=dev)
        o_nr = torch.zeros(1, dtype=torch.int32, device=dev)
        nnp.nnp_get_state(ctx, o_x, None, o_ep, None, o_nr)
        nnp.nnp_sync(ctx)
        xs = o_x.cpu().numpy().astype(np.float64)
        assert int(o_nr.item()) >= 2                       # the displacement rule fired at least once
        ref = orc.energy_forces(om, sp, xs, box, nbr_method=1)
        # potential energy of the last MD step (computed from the possibly stale-but-valid skinned lists)
        assert abs(float(o_ep.item()) - ref["E"][0]) <= U.E_RTOL * abs(ref["E"][0])
        # forces at the same positions, through the lists the MD loop would use next
        Eg, Fg = U.gpu_energy_forces(ctx, sp, xs, box, skin=0.5)
        U.assert_parity(Eg, Fg, ref)
    finally:
        nnp.nnp_destroy(ctx)


def test_full_config4_mixed_solvated(model1):
    consts, widths, params, om = model1
    sp, xyz, box = inputs.solvated_chain()
    assert len(np.unique(sp)) == 7 and len(sp) > 20000
    ctx = U.gpu_create(consts, widths, params, 1, len(sp))
    try:
        Eg, Fg = U.gpu_energy_forces(ctx, sp, xyz, box)
        _sampled_lists(ctx, xyz, box, len(sp), 0.0)
        U.assert_parity(Eg, Fg, orc.energy_forces(om, sp, xyz, box, nbr_method=1))
        assert nnp.nnp_aev_active_columns(ctx) == 1008
    finally:
        nnp.nnp_destroy(ctx)


def test_full_config5_molecule_batch8192():
    consts, widths, params, om = U.make_model(8, seed=inputs.SEED0 + 5)
    sp, xyz, offs = inputs.molecule_batch()
    n_mols = len(offs) - 1
    assert n_mols == 8192
    mol = np.repeat(np.arange(n_mols), np.diff(offs)).astype(np.int32)
    ctx = U.gpu_create(consts, widths, params, 8, len(sp), max_mols=n_mols)
    try:
        Eg, Fg = U.gpu_energy_forces(ctx, sp, xyz, None, mol_offsets=offs)
        _sampled_lists(ctx, xyz, None, len(sp), 0.0, mol_id=mol, n_sample=3000)
        ref = orc.energy_forces(om, sp, xyz, None, offs, want_e_atom=True)
        U.assert_parity(Eg, Fg, ref, mol_offsets=offs)
        strict, floor = U.assert_strict_energy_bar_where_it_is_defined(Eg, ref, offs)
        assert strict > 500      # the plain 1e-5 relative bar is what most of the 8192 molecules are held to
    finally:
        nnp.nnp_destroy(ctx)


# ---------------------------------------------------------------- active-column layout == dense layout
def test_dense_aev_layout_gives_the_same_result(model1):
    consts, widths, params, om = model1
    sp, xyz, box = inputs.water_box(216, seed=21)
    res = []
    for dense in (0, 1):
        p, keep = nnp.make_params(consts, widths, params, inputs.MASS, inputs.ACCEL_CONV, n_nets=1, mm_mode=U.MM_MODE,
                                  dense_aev=dense)
        ctx = nnp.nnp_create(p, len(sp), 1, 0, torch.cuda.current_stream().cuda_stream)
        try:
            res.append(U.gpu_energy_forces(ctx, sp, xyz, box))
            assert nnp.nnp_aev_active_columns(ctx) == (1008 if dense else 128)
            d_aev = torch.zeros((len(sp), 1008), dtype=torch.float32, device="cuda")
            nnp.nnp_get_aev(ctx, d_aev)
            nnp.nnp_sync(ctx)
            res[-1] = res[-1] + (d_aev.cpu().numpy(),)
        finally:
            nnp.nnp_destroy(ctx)
    ref = orc.energy_forces(om, sp, xyz, box)
    for Eg, Fg, _ in res:
        U.assert_parity(Eg, Fg, ref)
    assert np.array_equal(res[0][2], res[1][2])            # same AEV, column for column
    assert abs(res[0][0][0] - res[1][0][0]) <= 2e-6 * abs(ref["E"][0])
    # the same context re-laid out when the species set changes (H,O -> all seven -> H,O)
    ctx = U.gpu_create(consts, widths, params, 1, 4000)
    try:
        E1, F1 = U.gpu_energy_forces(ctx, sp, xyz, box)
        sp7, xyz7, box7 = inputs.solvated_chain(n_solute=300, L=22.0, seed=6)
        sp7 = sp7.copy(); sp7[:14] = np.arange(14) % 7
        E7, F7 = U.gpu_energy_forces(ctx, sp7, xyz7, box7)
        U.assert_parity(E7, F7, orc.energy_forces(om, sp7, xyz7, box7, nbr_method=1))
        E2, F2 = U.gpu_energy_forces(ctx, sp, xyz, box)
        assert E1[0] == E2[0] or abs(E1[0] - E2[0]) <= 1e-6 * abs(E1[0])
        U.assert_parity(E2, F2, ref)
    finally:
        nnp.nnp_destroy(ctx)


# ---------------------------------------------------------------- Gaussian ladder vs direct evaluation of the shift sets
@pytest.mark.parametrize("shifts", ["ani2x_direct", "nonuniform"])
def test_direct_shift_evaluation(model1, shifts, monkeypatch):
    """The default path evaluates the uniformly spaced ANI-2x shifts by the ladder recurrence (all other tests);
    here the direct evaluation: forced for the same constants, and chosen automatically for a non-uniform shift set."""
    consts, widths, params, om = model1
    if shifts == "ani2x_direct":
        monkeypatch.setenv("NNP_NO_LADDER", "1")
    else:
        rng = np.random.default_rng(77)
        consts = dict(consts)
        consts["shf_r"] = np.float32(consts["shf_r"] + rng.uniform(-0.05, 0.05, 16)).astype(np.float64)
        consts["shf_a"] = np.float32(consts["shf_a"] + rng.uniform(-0.05, 0.05, 8)).astype(np.float64)
        om = orc.OracleModel(consts, widths, params, 1)
    sp, xyz, box = inputs.solvated_chain(n_solute=300, L=22.0, seed=9)
    sp = sp.copy(); sp[:14] = np.arange(14) % 7
    ctx = U.gpu_create(consts, widths, params, 1, len(sp))
    try:
        assert nnp.nnp_aev_ladder(ctx) == 0
        Eg, Fg = U.gpu_energy_forces(ctx, sp, xyz, box)
        U.assert_parity(Eg, Fg, orc.energy_forces(om, sp, xyz, box, nbr_method=1))
    finally:
        nnp.nnp_destroy(ctx)


def test_ladder_is_the_default_for_ani2x_constants(model1):
    consts, widths, params, om = model1
    ctx = U.gpu_create(consts, widths, params, 1, 64)
    try:
        assert nnp.nnp_aev_ladder(ctx) == 1
    finally:
        nnp.nnp_destroy(ctx)


# ---------------------------------------------------------------- NEXT-1: Langevin BAOAB
@pytest.mark.parametrize("graph", [False, True], ids=["kernel_by_kernel", "cuda_graph"])
def test_langevin_baoab_against_oracle(model1, graph):
    consts, widths, params, om = model1
    sp, xyz, box = inputs.water_box(216, seed=19)
    v = inputs.maxwell_boltzmann(sp, 300.0, seed=4)
    n = len(sp)
    dt, gamma, kT, seed = 0.5, 0.02, inputs.KB * 300.0, 987654321012345
    dev = torch.device("cuda:0")
    ctx = U.gpu_create(consts, widths, params, 1, n, stream=torch.cuda.Stream(device=dev) if graph else None)
    try:
        d_sp = torch.as_tensor(sp, device=dev)
        d_x = torch.as_tensor(xyz.astype(np.float32), device=dev)
        d_v = torch.as_tensor(v.astype(np.float32), device=dev)
        o_x, o_v = torch.zeros_like(d_x), torch.zeros_like(d_v)
        o_ek = torch.zeros(1, dtype=torch.float64, device=dev)
        torch.cuda.synchronize()
        nnp.nnp_set_system(ctx, n, d_sp, d_x, box)
        with pytest.raises(nnp.NnpError):
            nnp.nnp_md_set_langevin(ctx, gamma, kT, seed)        # before nnp_md_init
        nnp.nnp_md_init(ctx, d_v, dt, 0.5)
        nnp.nnp_md_set_langevin(ctx, gamma, kT, seed)

        def state():
            nnp.nnp_get_state(ctx, o_x, o_v, None, o_ek, None)
            nnp.nnp_sync(ctx)
            return o_x.cpu().numpy().astype(np.float64), o_v.cpu().numpy().astype(np.float64), float(o_ek.item())

        # one step, then five more in one call (the device-side step counter feeds the generator)
        nnp.nnp_md_step(ctx, 1)
        x1, v1, _ = state()
        o1 = orc.md_langevin(om, sp, xyz, v, inputs.MASS, box, dt, inputs.ACCEL_CONV, 1, gamma, kT, seed)
        assert np.abs(x1 - o1["xyz"]).max() < 2e-6 and np.abs(v1 - o1["vel"]).max() < 2e-6
        kick = orc.md(om, sp, xyz, v, inputs.MASS, box, dt, inputs.ACCEL_CONV, 1)
        assert np.abs(v1 - kick["vel"]).max() > 1e-4             # the noise is in
        nnp.nnp_md_step(ctx, 5)
        x6, v6, ek6 = state()
        o6 = orc.md_langevin(om, sp, xyz, v, inputs.MASS, box, dt, inputs.ACCEL_CONV, 6, gamma, kT, seed)
        assert np.abs(x6 - o6["xyz"]).max() < 2e-5 and np.abs(v6 - o6["vel"]).max() < 2e-5
        assert abs(ek6 - o6["ekin"][6]) < 1e-4 * o6["ekin"][6]
        # gamma = 0 switches back to velocity Verlet: one step from the current state equals the oracle's VV step
        nnp.nnp_md_set_langevin(ctx, 0.0, kT, seed)
        nnp.nnp_md_step(ctx, 1)
        x7, v7, _ = state()
        o7 = orc.md(om, sp, x6, v6, inputs.MASS, box, dt, inputs.ACCEL_CONV, 1)
        assert np.abs(x7 - o7["xyz"]).max() < 2e-6 and np.abs(v7 - o7["vel"]).max() < 2e-6
    finally:
        nnp.nnp_destroy(ctx)


def test_langevin_thermostat_holds_temperature(model1):
    """648 atoms started at rest under random-weight forces (scale FORCE_SCALE_MD): friction 0.05/fs pulls the kinetic
    temperature to the bath's 300 K and holds it there."""
    consts, widths, _, _ = model1
    params = inputs.make_weights(inputs.SEED0, 1, last_layer_scale=inputs.FORCE_SCALE_MD)
    sp, xyz, box = inputs.water_box(216, seed=23)
    n = len(sp)
    dev = torch.device("cuda:0")
    ctx = U.gpu_create(consts, widths, params, 1, n, stream=torch.cuda.Stream(device=dev))
    try:
        d_sp = torch.as_tensor(sp, device=dev)
        d_x = torch.as_tensor(xyz.astype(np.float32), device=dev)
        d_v = torch.zeros_like(d_x)
        o_ek = torch.zeros(1, dtype=torch.float64, device=dev)
        torch.cuda.synchronize()
        nnp.nnp_set_system(ctx, n, d_sp, d_x, box)
        nnp.nnp_md_init(ctx, d_v, 0.5, 0.5)
        nnp.nnp_md_set_langevin(ctx, 0.05, inputs.KB * 300.0, 42)
        nnp.nnp_md_step(ctx, 400)
        temps = []
        for _ in range(40):
            nnp.nnp_md_step(ctx, 25)
            nnp.nnp_get_state(ctx, None, None, None, o_ek, None)
            nnp.nnp_sync(ctx)
            temps.append(2 * float(o_ek.item()) / (3 * n * inputs.KB))
        assert abs(np.mean(temps) - 300.0) < 20.0, np.mean(temps)
    finally:
        nnp.nnp_destroy(ctx)


# ---------------------------------------------------------------- NEXT-2: virial
VIRIAL_RTOL = 1e-5   # of sum |d_a (dE/dd)_b|, the scale the fp32 sums work at (the tensor itself is their cancelling sum)


def _gpu_virial(ctx, sp, xyz, box, skin=0.0, mol_offsets=None):
    dev = torch.device("cuda:0")
    n = len(sp)
    d_sp = torch.as_tensor(np.asarray(sp, dtype=np.int32), device=dev)
    d_x = torch.as_tensor(np.asarray(xyz, dtype=np.float32), device=dev).contiguous()
    n_mols = 1 if mol_offsets is None else len(mol_offsets) - 1
    d_mo = None if mol_offsets is None else torch.as_tensor(np.asarray(mol_offsets, dtype=np.int32), device=dev)
    d_E = torch.zeros(n_mols, dtype=torch.float64, device=dev)
    d_F = torch.zeros((n, 3), dtype=torch.float32, device=dev)
    d_V = torch.zeros(9, dtype=torch.float64, device=dev)
    torch.cuda.synchronize()
    nnp.nnp_set_system(ctx, n, d_sp, d_x, box, n_mols, d_mo)
    nnp.nnp_build_neighbors(ctx, skin)
    nnp.nnp_energy_forces_virial(ctx, d_E, d_F, d_V)
    nnp.nnp_sync(ctx)
    return d_E.cpu().numpy(), d_F.cpu().numpy().astype(np.float64), d_V.cpu().numpy().reshape(3, 3)


@pytest.mark.parametrize("system", ["water_periodic_skin", "mixed_periodic", "molecule"])
def test_virial_against_oracle(model1, system):
    consts, widths, params, om = model1
    skin = 0.0
    if system == "water_periodic_skin":
        sp, xyz, box = inputs.water_box(1000, seed=41)
        skin = 0.5                                         # entries beyond the cutoff must contribute nothing
    elif system == "mixed_periodic":
        sp, xyz, box = inputs.solvated_chain(n_solute=300, L=22.0, seed=43)
        sp = sp.copy(); sp[:14] = np.arange(14) % 7
    else:
        sp, xyz, _ = inputs.molecule_batch(1, nmin=30, nmax=30, seed=45)
        box = None
    ctx = U.gpu_create(consts, widths, params, 1, len(sp))
    try:
        Eg, Fg, Vg = _gpu_virial(ctx, sp, xyz, box, skin)
        ref = orc.energy_forces_virial(om, sp, xyz, box, nbr_method=1 if box is not None else 0)
        U.assert_parity(Eg, Fg, ref)
        assert np.abs(Vg - ref["virial"]).max() <= VIRIAL_RTOL * ref["virial_abs"], (Vg, ref["virial"])
        assert np.array_equal(Vg, Vg.T)
        if box is None:                                    # Clausius form from the GPU's own forces
            assert np.abs(Vg + xyz.T @ Fg).max() <= 3 * VIRIAL_RTOL * ref["virial_abs"]
        # the plain entry point still gives the same energy and forces
        E2, F2 = U.gpu_energy_forces(ctx, sp, xyz, box, skin=skin)
        assert abs(E2[0] - Eg[0]) <= 1e-6 * abs(Eg[0]) and np.abs(F2 - Fg).max() < 1e-4
    finally:
        nnp.nnp_destroy(ctx)


def test_virial_needs_a_single_structure(model1):
    consts, widths, params, om = model1
    sp, xyz, offs = inputs.molecule_batch(3, seed=46)
    ctx = U.gpu_create(consts, widths, params, 1, len(sp), max_mols=3)
    try:
        with pytest.raises(nnp.NnpError):
            _gpu_virial(ctx, sp, xyz, None, mol_offsets=offs)
    finally:
        nnp.nnp_destroy(ctx)


def test_measured_peaks_are_plausible():
    """nnp_measure_peaks: the micro-benchmarks run and land in the range the hardware allows.
    B200: 148 SMs x 128 FMA lanes x 2 x 1.965 GHz = 74.4 TFLOP/s fp32, 148 x 16 x 1.965 GHz = 4.65 T MUFU ops/s, dense
    TF32 tcgen05 nominally half of bf16 (2.25 PFLOP/s)."""
    pk = nnp.nnp_measure_peaks(0)
    assert 30.0 < pk["fp32_fma_tflops"] < 80.0, pk
    assert 1500.0 < pk["mufu_ex2_gops"] < 5000.0, pk
    for form in ("ss", "ts"):
        assert 300.0 < pk["tf32_tcgen05_%s_tflops" % form] < 1300.0, pk
        assert 16.0 <= pk["cycles_per_mma_m128n256k8_%s" % form] < 400.0, pk


# ---------------------------------------------------------------- SURVEY 8(f)-2, second part: general cells, all periodic images
def _lists_outside_guard_band(ctx, xyz, cell, n, skin, band=2e-4):
    """fp64 all-images lists of the oracle against the rows of the caller's atoms (an image of j is reported as j): equal
    as multisets once the pairs within `band` of the list radius - where fp32 and fp64 may disagree - are set aside."""
    for which, rc in ((0, 5.1), (1, 3.5)):
        rl = float(np.float32(rc) + np.float32(skin))
        got = U.gpu_neighbors(ctx, which, n, stride=640)
        inner = orc.neighbors_cell(xyz, cell, rl - band)
        outer = orc.neighbors_cell(xyz, cell, rl + band)
        for i in range(n):
            g = sorted(int(j) for j in got[i])
            lo, hi = sorted(j for j, *_ in inner[i]), sorted(j for j, *_ in outer[i])
            assert len(lo) <= len(g) <= len(hi), (which, i, len(lo), len(g), len(hi))
            from collections import Counter
            cg, cl, ch = Counter(g), Counter(lo), Counter(hi)
            assert all(cg[j] >= cl[j] for j in cl) and all(ch[j] >= cg[j] for j in cg), (which, i)


VIRIAL_RTOL_CELL = 1e-5


def test_triclinic_cell_against_oracle(model1):
    """A sheared 343-water cell (perpendicular widths 20.8 / 19.6 / 22.7 A: minimum image, fractional-coordinate bins):
    lists, energy, forces and the full virial against the oracle's all-images definition; unwrapped coordinates; then one
    and ten MD steps against the oracle's integrator in the same cell."""
    consts, widths, params, om = model1
    sp, x0, box = inputs.water_box(343, seed=61)
    D = np.array([[1.0, 0.0, 0.0], [0.21, 0.94, 0.0], [-0.13, 0.17, 1.05]])
    cell = (np.diag(box) @ D).astype(np.float32).astype(np.float64)
    rng = np.random.default_rng(1)
    xyz = (x0 @ D + rng.integers(-2, 3, size=(len(sp), 3)) @ cell).astype(np.float32).astype(np.float64)
    n = len(sp)
    dev = torch.device("cuda:0")
    ctx = U.gpu_create(consts, widths, params, 1, n)
    try:
        Eg, Fg, Vg = U.gpu_energy_forces_cell(ctx, sp, xyz, cell, skin=0.3, want_virial=True)
        _lists_outside_guard_band(ctx, xyz, cell, n, 0.3)
        ref = orc.energy_forces_cell(om, sp, xyz, cell, want_virial=True)
        U.assert_parity(Eg, Fg, ref)
        assert np.abs(Vg - ref["virial"]).max() <= VIRIAL_RTOL_CELL * ref["virial_abs"], (Vg, ref["virial"])
        # MD in the triclinic cell
        v = inputs.maxwell_boltzmann(sp, 300.0, seed=5).astype(np.float32).astype(np.float64)
        d_v = torch.as_tensor(v.astype(np.float32), device=dev)
        nnp.nnp_md_init(ctx, d_v, 0.5, 0.5)
        o_x, o_v = torch.zeros((n, 3), device=dev), torch.zeros((n, 3), device=dev)
        o_ep, o_ek = torch.zeros(1, dtype=torch.float64, device=dev), torch.zeros(1, dtype=torch.float64, device=dev)
        nnp.nnp_md_step(ctx, 1)
        nnp.nnp_get_state(ctx, o_x, o_v, o_ep, o_ek, None)
        nnp.nnp_sync(ctx)
        o1 = orc.md_cell(om, sp, xyz, v, inputs.MASS, cell, 0.5, inputs.ACCEL_CONV, 1)
        assert np.abs(o_x.cpu().numpy() - o1["xyz"]).max() < 1e-5 and np.abs(o_v.cpu().numpy() - o1["vel"]).max() < 2e-6
        assert abs(float(o_ep.item()) - o1["epot"][1]) <= 2e-5 * abs(o1["epot"][1])
        nnp.nnp_md_step(ctx, 30)
        nnp.nnp_get_state(ctx, o_x, o_v, o_ep, o_ek, None)
        nnp.nnp_sync(ctx)
        xs = o_x.cpu().numpy().astype(np.float64)
        r2 = orc.energy_forces_cell(om, sp, xs, cell, want_forces=False)
        assert abs(float(o_ep.item()) - r2["E"][0]) <= U.E_RTOL * abs(r2["E"][0])
    finally:
        nnp.nnp_destroy(ctx)


@pytest.mark.parametrize("case", ["cubic_9.31", "cubic_4.9_below_the_cutoff", "triclinic_small"])
def test_small_cells_see_all_periodic_images(model1, case):
    """Cells narrower than 2 (rcr + skin), down to one smaller than the cutoff (atoms see their own images and several
    images of one neighbour): energy per cell, forces, virial and the rows of the caller's atoms against the oracle's
    explicit sum over images.  The library evaluates the smallest supercell that allows the minimum image."""
    consts, widths, params, om = model1
    if case == "cubic_9.31":
        sp, xyz, box = inputs.water_box(27, 9.31, seed=3)
        cell, copies = np.diag(box).astype(np.float64), 8
    elif case == "cubic_4.9_below_the_cutoff":
        sp, xyz, box = inputs.water_box(4, 4.9, seed=4)
        cell, copies = np.diag(box).astype(np.float64), 27
    else:
        sp, x0, box = inputs.water_box(8, 6.2, seed=6)
        D = np.array([[1.0, 0.0, 0.0], [0.23, 0.94, 0.0], [-0.17, 0.12, 1.05]])
        cell = (np.diag(box) @ D).astype(np.float32).astype(np.float64)
        xyz = (x0 @ D).astype(np.float32).astype(np.float64)
        copies = 8
    n = len(sp)
    ctx = U.gpu_create(consts, widths, params, 1, n * copies, cap_r=320, cap_a=128)
    try:
        Eg, Fg, Vg = U.gpu_energy_forces_cell(ctx, sp, xyz, cell, want_virial=True)
        ref = orc.energy_forces_cell(om, sp, xyz, cell, want_virial=True)
        U.assert_parity(Eg, Fg, ref)
        assert np.abs(Vg - ref["virial"]).max() <= VIRIAL_RTOL_CELL * ref["virial_abs"], (Vg, ref["virial"])
        _lists_outside_guard_band(ctx, xyz, cell, n, 0.0)
        # AEV rows of the caller's atoms
        d_aev = torch.zeros((n, 1008), dtype=torch.float32, device="cuda")
        nnp.nnp_get_aev(ctx, d_aev)
        nnp.nnp_sync(ctx)
        aev_ref = orc.energy_forces_cell(om, sp, xyz, cell, want_forces=False, want_aev=True)["aev"]
        assert np.abs(d_aev.cpu().numpy() - aev_ref).max() < 2e-5 * max(1.0, np.abs(aev_ref).max())
        # MD: every internal copy follows its atom; against the oracle's integrator in the small cell (all images)
        v = inputs.maxwell_boltzmann(sp, 300.0, seed=8).astype(np.float32).astype(np.float64)
        dev = torch.device("cuda:0")
        nnp.nnp_md_init(ctx, torch.as_tensor(v.astype(np.float32), device=dev), 0.5, 0.3)
        o_x, o_v = torch.zeros((n, 3), device=dev), torch.zeros((n, 3), device=dev)
        o_ep, o_ek = torch.zeros(1, dtype=torch.float64, device=dev), torch.zeros(1, dtype=torch.float64, device=dev)
        nnp.nnp_md_step(ctx, 3)
        nnp.nnp_get_state(ctx, o_x, o_v, o_ep, o_ek, None)
        nnp.nnp_sync(ctx)
        o3 = orc.md_cell(om, sp, xyz, v, inputs.MASS, cell, 0.5, inputs.ACCEL_CONV, 3)
        assert np.abs(o_x.cpu().numpy() - o3["xyz"]).max() < 1e-5 and np.abs(o_v.cpu().numpy() - o3["vel"]).max() < 1e-5
        assert abs(float(o_ep.item()) - o3["epot"][3]) <= 2e-5 * abs(o3["epot"][3])
        assert abs(float(o_ek.item()) - o3["ekin"][3]) <= 1e-4 * o3["ekin"][3]
        nnp.nnp_md_step(ctx, 40)
        nnp.nnp_get_state(ctx, o_x, o_v, o_ep, o_ek, None)
        nnp.nnp_sync(ctx)
        r2 = orc.energy_forces_cell(om, sp, o_x.cpu().numpy().astype(np.float64), cell, want_forces=False)
        assert abs(float(o_ep.item()) - r2["E"][0]) <= U.E_RTOL * abs(r2["E"][0])
    finally:
        nnp.nnp_destroy(ctx)
    # a context too small for the supercell says so
    ctx = U.gpu_create(consts, widths, params, 1, n)
    try:
        with pytest.raises(nnp.NnpError) as e:
            U.gpu_energy_forces_cell(ctx, sp, xyz, cell)
        assert e.value.status == nnp.NNP_EBOX
    finally:
        nnp.nnp_destroy(ctx)


@pytest.mark.parametrize("n_present", [3, 4, 5, 6], ids=["256_columns", "384_columns", "576_columns", "768_columns"])
def test_fused_chain_on_every_number_of_active_columns(model1, n_present):
    """The fused chain streams its first and last GEMM in passes of 256 columns when the loaded system has more active AEV
    columns than a TMEM region holds: 3 species present = 256 columns (the widest single pass), 4 = 384 (passes 256 + 128,
    input passes of 16 + 8 chunks), 5 = 576 (256 + 256 + 64; 16 + 16 + 4), 6 = 768; two networks, so the output passes add
    into dE/dG with reductions.  Water (128) and all seven species (1024) are covered by the other tests."""
    consts, widths, params, om = U.make_model(2, seed=inputs.SEED0 + 77)
    sp, xyz, box = inputs.solvated_chain(n_solute=500, L=22.0, seed=9)
    sp = sp.copy()
    sp[:14] = np.arange(14) % 7
    sp = np.minimum(sp, n_present - 1).astype(sp.dtype)      # species >= n_present become the last one present
    assert len(np.unique(sp)) == n_present
    ctx = U.gpu_create(consts, widths, params, 2, len(sp))
    try:
        Eg, Fg = U.gpu_energy_forces(ctx, sp, xyz, box)
        assert nnp.nnp_aev_active_columns(ctx) == n_present * 16 + n_present * (n_present + 1) // 2 * 32
        ref = orc.energy_forces(om, sp, xyz, box, nbr_method=1, want_e_atom=True)
        U.assert_parity(Eg, Fg, ref)
        # twice more on the same context: the results of the chain do not depend on timing (a ring-buffer phase bug once did)
        for _ in range(2):
            E2, F2 = U.gpu_energy_forces(ctx, sp, xyz, box)
            assert abs(E2[0] - Eg[0]) <= 2e-7 * np.abs(ref["e_atom"]).sum() and np.abs(F2 - Fg).max() < 2e-4
    finally:
        nnp.nnp_destroy(ctx)
