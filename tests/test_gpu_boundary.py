"""-m gpu tests of the boundary and of the paths no workload of the paper reaches: allocator hooks, graph
re-capture after a public nnp_build_neighbors, the non-default matmul modes at their own bars, dense systems
(neighbour capacities, the reverse kernel's fallback), element-wise AEV parity for all seven species."""
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


# ---------------------------------------------------------------- device memory through the caller's allocator
def test_allocator_hooks_with_the_torch_caching_allocator(model1):
    """Every device buffer of the library comes from nnp_params.alloc: here torch.cuda.caching_allocator_alloc, so the
    library's scratch is accounted for (and recycled) by PyTorch.  Parity is unchanged; every block is handed back."""
    consts, widths, params, om = model1
    sp, xyz, box = inputs.water_box(64, 12.42)
    live, stats = {}, {"alloc": 0, "free": 0, "bytes": 0}
    stream = torch.cuda.current_stream()

    def alloc(nbytes, user):
        ptr = torch.cuda.caching_allocator_alloc(int(nbytes), 0, stream)
        live[ptr] = nbytes
        stats["alloc"] += 1
        stats["bytes"] += nbytes
        return ptr

    def dealloc(ptr, user):
        assert ptr in live
        del live[ptr]
        stats["free"] += 1
        torch.cuda.caching_allocator_delete(ptr)

    before = torch.cuda.memory_allocated()
    p, keep = nnp.make_params(consts, widths, params, inputs.MASS, inputs.ACCEL_CONV, n_nets=1, mm_mode=U.MM_MODE,
                              alloc=alloc, dealloc=dealloc)
    ctx = nnp.nnp_create(p, len(sp), 1, 0, stream.cuda_stream)
    try:
        assert stats["alloc"] >= 30 and len(live) == stats["alloc"]
        assert torch.cuda.memory_allocated() - before >= stats["bytes"]       # torch accounts for the library's memory
        Eg, Fg = U.gpu_energy_forces(ctx, sp, xyz, box)
        U.assert_parity(Eg, Fg, orc.energy_forces(om, sp, xyz, box))
        # a second, larger grid (more keys) re-allocates the cell arrays through the same hooks
        sp2, xyz2, box2 = inputs.water_box(64, 40.0, seed=3)
        Eg2, Fg2 = U.gpu_energy_forces(ctx, sp2, xyz2, box2)
        U.assert_parity(Eg2, Fg2, orc.energy_forces(om, sp2, xyz2, box2))
    finally:
        nnp.nnp_destroy(ctx)
    assert not live and stats["free"] == stats["alloc"]
    assert torch.cuda.memory_allocated() == before
    # alloc without dealloc is rejected
    p2, keep2 = nnp.make_params(consts, widths, params, inputs.MASS, inputs.ACCEL_CONV, alloc=alloc, dealloc=dealloc)
    p2.dealloc = nnp.DEALLOC_FN()
    with pytest.raises(nnp.NnpError):
        nnp.nnp_create(p2, 8, 1, 0, stream.cuda_stream)


# ---------------------------------------------------------------- nnp_build_neighbors while an MD graph exists
def test_build_neighbors_between_md_steps_recaptures_the_graph(model1, monkeypatch):
    """A public nnp_build_neighbors with another skin between nnp_md_step calls: the captured step graph (which has the
    skin, the grid and the key arrays baked in) is dropped and re-captured; the trajectory equals the kernel-by-kernel
    path's (NNP_NO_GRAPH=1) and the lists are the new skin's."""
    consts, widths, params, om = model1
    sp, xyz, box = inputs.water_box(216, seed=31)
    v = inputs.maxwell_boltzmann(sp, 300.0, seed=5)
    n = len(sp)
    dev = torch.device("cuda:0")
    out = []
    for no_graph in ("0", "1"):
        monkeypatch.setenv("NNP_NO_GRAPH", no_graph)
        ctx = U.gpu_create(consts, widths, params, 1, n, stream=torch.cuda.Stream(device=dev))
        try:
            d_sp = torch.as_tensor(sp, device=dev)
            d_x = torch.as_tensor(xyz.astype(np.float32), device=dev)
            d_v = torch.as_tensor(v.astype(np.float32), device=dev)
            torch.cuda.synchronize()
            nnp.nnp_set_system(ctx, n, d_sp, d_x, box)
            nnp.nnp_md_init(ctx, d_v, 0.5, 0.5)
            nnp.nnp_md_step(ctx, 4)
            nnp.nnp_build_neighbors(ctx, 0.9)      # another skin: other list radii, half-skin threshold and cell grid
            nnp.nnp_md_step(ctx, 4)
            o_x, o_v = torch.zeros_like(d_x), torch.zeros_like(d_v)
            nnp.nnp_get_state(ctx, o_x, o_v, None, None, None)
            nnp.nnp_sync(ctx)
            xs = o_x.cpu().numpy().astype(np.float64)
            got = U.gpu_neighbors(ctx, 0, n)
            out.append((xs, o_v.cpu().numpy().astype(np.float64), got))
        finally:
            nnp.nnp_destroy(ctx)
    (xa, va, la), (xb, vb, lb) = out
    assert np.abs(xa - xb).max() < 5e-6 and np.abs(va - vb).max() < 5e-6
    # the rows of the graph path are lists with the NEW skin (built at some earlier positions: supersets of the exact
    # 5.1 A lists at the final positions, subsets of the 5.1 + 0.9 + 2 * 0.45 ones)
    inner = orc.neighbors(xa, box, 5.1, fp32_pred=True, method="grid")
    outer = orc.neighbors(xa, box, 5.1 + 0.9 + 0.9, fp32_pred=True, method="grid")
    for i in range(n):
        assert set(inner[i]) <= set(la[i]) <= set(outer[i])
    # (6.0 / 5.1)^3 = 1.63: the rows are visibly longer than cutoff rows (and than 0.5 A-skin rows, 1.32): the new skin is in use
    assert sum(len(r) for r in la) > 1.45 * sum(len(r) for r in inner)


# ---------------------------------------------------------------- the matmul modes at their own bars
def _errors(mm_mode, consts, widths, params, om, sp, xyz, box):
    ctx = U.gpu_create(consts, widths, params, 1, len(sp), mm_mode=mm_mode)
    try:
        Eg, Fg = U.gpu_energy_forces(ctx, sp, xyz, box)
    finally:
        nnp.nnp_destroy(ctx)
    ref = orc.energy_forces(om, sp, xyz, box, nbr_method=1)
    return abs(Eg[0] - ref["E"][0]) / abs(ref["E"][0]), np.abs(Fg - ref["F"]).max()


def test_matmul_modes_at_their_own_bars(model1):
    """PAPER.md L315-321 (Fig. 3): only fp32-grade matmuls are acceptable, TF32 is not.  Plain TF32 (mm_mode 2) is a public
    mode: it must run, land at the order DESIGN.md section 6 states (|dE|/|E| ~ 2e-4, max |dF| ~ 3e-2 at RMS F ~ 20) and
    FAIL the fp32 bars; 3xTF32, fp32 SIMT and the fp64-accumulate leg meet them, in that order of accuracy."""
    consts, widths, params, om = model1
    sp, xyz, box = inputs.water_box(343, seed=51)
    err = {m: _errors(m, consts, widths, params, om, sp, xyz, box)
           for m in (nnp.NNP_MM_FP32_SIMT, nnp.NNP_MM_3XTF32_TC, nnp.NNP_MM_TF32_TC, nnp.NNP_MM_FP64_SIMT, nnp.NNP_MM_3XF16_TC)}
    print("mode: (|dE|/|E|, max|dF|)", err)
    for m in (nnp.NNP_MM_FP32_SIMT, nnp.NNP_MM_3XTF32_TC, nnp.NNP_MM_FP64_SIMT, nnp.NNP_MM_3XF16_TC):
        assert err[m][0] <= U.E_RTOL and err[m][1] <= U.F_ATOL, (m, err[m])
    # the fp16 hi/lo split carries the same 11 + 11 bits as the tf32 split: the two fp32-grade tensor-core modes land together
    assert err[nnp.NNP_MM_3XF16_TC][1] <= 3.0 * err[nnp.NNP_MM_3XTF32_TC][1] + 1e-5
    e2, f2 = err[nnp.NNP_MM_TF32_TC]
    assert e2 < 5e-3 and f2 < 0.3, (e2, f2)                       # its own, looser bar: the right order of magnitude
    assert f2 > U.F_ATOL                                           # ... and it does NOT meet the fp32 force bar
    assert f2 > 20 * err[nnp.NNP_MM_3XTF32_TC][1]
    # the fp64-accumulate contraction is at least as good as fp32 FMA (what is left is the fp32 AEV and storage rounding)
    assert err[nnp.NNP_MM_FP64_SIMT][1] <= 1.5 * err[nnp.NNP_MM_FP32_SIMT][1] + 1e-6


def test_tf32_mode_md_runs_and_ensemble(model1):
    """k_gemm_tc<*, false> through every epilogue: a 3-network ensemble (EPI_RED) and a few MD steps."""
    consts, widths, params, om = U.make_model(3, seed=inputs.SEED0 + 21)
    sp, xyz, box = inputs.water_box(216, seed=inputs.SEED0 + 22)
    ctx = U.gpu_create(consts, widths, params, 3, len(sp), mm_mode=nnp.NNP_MM_TF32_TC)
    try:
        Eg, Fg = U.gpu_energy_forces(ctx, sp, xyz, box)
        ref = orc.energy_forces(om, sp, xyz, box, want_e_atom=True)
        assert abs(Eg[0] - ref["E"][0]) <= 2e-3 * np.abs(ref["e_atom"]).sum()
        assert np.abs(Fg - ref["F"]).max() < 0.3
    finally:
        nnp.nnp_destroy(ctx)


# ---------------------------------------------------------------- AEV element by element, all seven species
def test_aev_elementwise_seven_species(model1):
    """Dense 1008-column layout, 28 species-pair blocks, the non-GS reverse kernel: G itself against the oracle, column for
    column (config 1's check covers only the 128 active columns of water)."""
    consts, widths, params, om = model1
    sp, xyz, box = inputs.solvated_chain(n_solute=600, L=24.0, seed=5)
    sp = sp.copy()
    sp[:14] = np.arange(14) % 7
    ctx = U.gpu_create(consts, widths, params, 1, len(sp))
    try:
        Eg, Fg = U.gpu_energy_forces(ctx, sp, xyz, box)
        assert nnp.nnp_aev_active_columns(ctx) == 1008
        d_aev = torch.zeros((len(sp), 1008), dtype=torch.float32, device="cuda")
        nnp.nnp_get_aev(ctx, d_aev)
        nnp.nnp_sync(ctx)
        ref = orc.energy_forces(om, sp, xyz, box, nbr_method=1, want_aev=True)
        got = d_aev.cpu().numpy()
        assert np.abs(got - ref["aev"]).max() < 2e-5 * max(1.0, np.abs(ref["aev"]).max())
        ang = ref["aev"][:, 112:].reshape(len(sp), 28, 32)
        assert (np.abs(ang).sum((0, 2)) > 0).sum() >= 20           # most of the 28 pair blocks are populated
        assert np.array_equal(got == 0, ref["aev"] == 0) or np.abs(got[ref["aev"] == 0]).max() < 1e-12
    finally:
        nnp.nnp_destroy(ctx)


# ---------------------------------------------------------------- dense systems: capacities and the reverse fallback
def test_dense_box_reverse_fallback_and_long_rows(model1):
    """0.25 atoms / A^3 (water: 0.10): 33-64 angular neighbours inside 3.5 A for most centres (the reverse kernel's pair
    arena covers 32: beyond it the shared-memory-atomics fallback runs), ~139 radial neighbours (more than the three
    prefetched trips), rows longer than 64 in the angular list (cap_a = 128: the extra-chunk loop).  E, F and the virial."""
    consts, widths, params, om = model1
    sp, xyz, box = inputs.dense_box(0.25)
    n = len(sp)
    ctx = U.gpu_create(consts, widths, params, 1, n, cap_r=320, cap_a=128)
    try:
        skin = 0.4
        dev = torch.device("cuda:0")
        d_E = torch.zeros(1, dtype=torch.float64, device=dev)
        d_F = torch.zeros((n, 3), dtype=torch.float32, device=dev)
        d_V = torch.zeros(9, dtype=torch.float64, device=dev)
        nnp.nnp_set_system(ctx, n, torch.as_tensor(sp, device=dev), torch.as_tensor(xyz.astype(np.float32), device=dev), box)
        nnp.nnp_build_neighbors(ctx, skin)
        nnp.nnp_energy_forces_virial(ctx, d_E, d_F, d_V)
        nnp.nnp_sync(ctx)
        for which, rc in ((0, 5.1), (1, 3.5)):
            got = U.gpu_neighbors(ctx, which, n, stride=320)
            ref = orc.neighbors(xyz, box, float(np.float32(rc) + np.float32(skin)), fp32_pred=True)
            assert all(np.array_equal(got[i], ref[i]) for i in range(n))
        n_in = np.array([len(r) for r in orc.neighbors(xyz, box, 3.5)])
        n_row = np.array([len(r) for r in orc.neighbors(xyz, box, float(np.float32(3.5) + np.float32(skin)), fp32_pred=True)])
        n_rad = np.array([len(r) for r in orc.neighbors(xyz, box, 5.1)])
        assert n_in.max() <= 64 and (n_in > 32).sum() > n // 2 and n_row.max() > 64 and n_rad.mean() > 120, \
            (n_in.min(), n_in.max(), n_row.max(), n_rad.mean())
        ref = orc.energy_forces_virial(om, sp, xyz, box)
        # forces here are ~5 times the water ones (RMS printed): the absolute 1e-3 bar is taken relative to that scale
        rms = np.sqrt((ref["F"] ** 2).sum(1).mean())
        Eg, Fg = d_E.cpu().numpy(), d_F.cpu().numpy().astype(np.float64)
        assert abs(Eg[0] - ref["E"][0]) <= U.E_RTOL * abs(ref["E"][0])
        assert np.abs(Fg - ref["F"]).max() <= U.F_ATOL * max(1.0, rms / 20.0), (np.abs(Fg - ref["F"]).max(), rms)
        Vg = d_V.cpu().numpy().reshape(3, 3)
        assert np.abs(Vg - ref["virial"]).max() <= 1e-5 * ref["virial_abs"]
    finally:
        nnp.nnp_destroy(ctx)


def test_more_than_64_angular_neighbours_in_cutoff_is_reported(model1):
    """0.42 atoms / A^3: ~75 atoms inside 3.5 A.  The rows fit (cap_a = 160), the 64 shared-memory slots of the AEV kernels
    do not: NNP_ECAPACITY, never a silently truncated sum (include/nnp.h, nnp_params.cap_a)."""
    consts, widths, params, om = model1
    sp, xyz, box = inputs.dense_box(0.42, dmin=1.0, seed=inputs.SEED0 + 8)
    n_in = np.array([len(r) for r in orc.neighbors(xyz, box, 3.5)])
    assert n_in.max() > 64
    ctx = U.gpu_create(consts, widths, params, 1, len(sp), cap_r=400, cap_a=160)
    try:
        with pytest.raises(nnp.NnpError) as e:
            U.gpu_energy_forces(ctx, sp, xyz, box)
        assert e.value.status == nnp.NNP_ECAPACITY
    finally:
        nnp.nnp_destroy(ctx)


def test_bad_mol_offsets_are_rejected(model1):
    consts, widths, params, om = model1
    ctx = U.gpu_create(consts, widths, params, 1, 16, max_mols=4)
    try:
        sp = np.zeros(6, np.int32)
        xyz = np.arange(18, dtype=np.float64).reshape(6, 3)
        for offs in ([0, 4, 2, 6], [1, 2, 4, 6], [0, 2, 4, 5]):
            with pytest.raises(nnp.NnpError) as e:
                U.gpu_energy_forces(ctx, sp, xyz, None, mol_offsets=offs)
            assert e.value.status == nnp.NNP_EINVAL
        U.gpu_energy_forces(ctx, sp, xyz, None, mol_offsets=[0, 2, 2, 6])      # an empty structure is fine
    finally:
        nnp.nnp_destroy(ctx)


def test_repeatability_stress():
    """The same structures evaluated again and again (water, 4 and 7 species, a molecule batch with an ensemble; default and
    side stream): any repeat that deviates beyond the noise of the fp32 force scatter fails.  This is the test that found the
    input-ring phase bug of the fused chain (rare wrong energies on seven-species systems)."""
    import sys
    from paper_2405_01491_b200 import repeatability
    argv = sys.argv
    sys.argv = ["repeatability", "--repeats", "20"]
    try:
        assert repeatability.main() == 0
    finally:
        sys.argv = argv

@pytest.mark.gpu
def test_buckets_of_more_than_32_atoms_are_ordered_too(model1):
    """The neighbour build orders every (species, cell) bucket by previous index: one warp ranks a bucket of up to 32 atoms,
    lane 0 sorts larger ones serially.  A dense one-species box (54 atoms per cell) and a non-periodic cluster of 150 atoms
    (its single "cell" is the structure) take that path; lists as exact rows, E and F against the oracle, and the same
    result on a second evaluation after the atoms have been re-sorted once more."""
    consts, widths, params, om = model1
    cases = []
    sp, xyz, box = inputs.dense_box(0.25, n_species=1)
    cases.append((sp, xyz, box, 320, 128))
    spw, xyzw, boxw = inputs.water_box(216)
    centre = xyzw.mean(0)
    keep = np.argsort(((xyzw - centre) ** 2).sum(1))[:150]
    cases.append((spw[keep].astype(np.int32), xyzw[keep], None, 160, 64))
    for sp, xyz, box, cap_r, cap_a in cases:
        n = len(sp)
        assert np.bincount(sp).max() > 32
        ctx = U.gpu_create(consts, widths, params, 1, n, cap_r=cap_r, cap_a=cap_a)
        try:
            ref = orc.energy_forces(om, sp, xyz, box)
            rms = np.sqrt((ref["F"] ** 2).sum(1).mean())
            for rep in range(2):
                Eg, Fg = U.gpu_energy_forces(ctx, sp, xyz, box)
                assert abs(Eg[0] - ref["E"][0]) <= U.E_RTOL * abs(ref["E"][0])
                assert np.abs(Fg - ref["F"]).max() <= U.F_ATOL * max(1.0, rms / 20.0)
            for which, rc in ((0, 5.1), (1, 3.5)):
                got = U.gpu_neighbors(ctx, which, n, stride=cap_r)
                want = orc.neighbors(xyz, box, float(np.float32(rc)), fp32_pred=True)
                assert all(np.array_equal(got[i], want[i]) for i in range(n))
        finally:
            nnp.nnp_destroy(ctx)

@pytest.mark.gpu
def test_cell_tiled_list_build_gives_the_defined_rows(model1, monkeypatch):
    """The one-block-per-cell list kernel tests wrapped, image-shifted coordinates and hands the candidates inside a guard
    band of a list radius to the defined fp32 predicate.  4096 waters, every atom moved by up to +-3 box lengths per
    dimension (unwrapped MD coordinates: the wrapped values then carry the rounding of the larger numbers): the rows of
    both kernels equal the oracle's fp32-predicate rows, with and without a skin."""
    consts, widths, params, om = model1
    sp, xyz, box = inputs.water_box(4096)
    rng = np.random.default_rng(11)
    xyz = (xyz + rng.integers(-3, 4, size=xyz.shape) * box).astype(np.float32).astype(np.float64)
    n = len(sp)
    for skin in (0.0, 0.5):
        want = [orc.neighbors(xyz, box, float(np.float32(rc) + np.float32(skin)), fp32_pred=True) for rc in (5.1, 3.5)]
        for tile in ("1", "0"):
            monkeypatch.setenv("NNP_LIST_TILE", tile)
            ctx = U.gpu_create(consts, widths, params, 1, n)
            try:
                U.gpu_energy_forces(ctx, sp, xyz, box, skin=skin)
                for which in (0, 1):
                    got = U.gpu_neighbors(ctx, which, n, stride=160)
                    bad = [i for i in range(n) if not np.array_equal(got[i], want[which][i])]
                    assert not bad, (tile, skin, which, len(bad), bad[:5])
            finally:
                nnp.nnp_destroy(ctx)



