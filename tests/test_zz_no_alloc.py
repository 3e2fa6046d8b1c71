"""-m gpu test of nnp_neighbors_no_alloc (include/nnp.h, csrc/no_alloc.cu): the neighbour lists built with the scratch memory
in the library's static device array against the existing path (nnp_build_neighbors + nnp_get_neighbors), whose rows the
parity tests pin to the oracle.  Index work: the rows must be equal as sets, exactly.  Collected last on purpose
(test_zz_...): the suite runs with pytest -x, a failure here must not hide another test."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from paper_2405_01491_b200 import inputs, nnp  # noqa: E402
from tests import gpu_util as U               # noqa: E402


def _rows_no_alloc(xyz, box, rcut, stride=160, stream=None):
    dev = torch.device("cuda:0")
    n = len(xyz)
    d_x = torch.as_tensor(np.asarray(xyz, dtype=np.float32), device=dev).contiguous()
    d_c = torch.full((max(n, 1),), -7, dtype=torch.int32, device=dev)
    d_l = torch.full((max(n, 1), stride), -1, dtype=torch.int32, device=dev)
    torch.cuda.synchronize()
    nnp.nnp_neighbors_no_alloc(n, d_x, box, rcut, d_c, d_l, stride, stream)
    torch.cuda.synchronize()
    c, l = d_c.cpu().numpy(), d_l.cpu().numpy()
    assert (c[:n] >= 0).all() and c[:n].max() <= stride
    return [np.sort(l[i, :c[i]]) for i in range(n)]


def _rows_existing(model, species, xyz, box, skin):
    """The existing path: radial list (rcr = 5.1 A) with a skin, i.e. radius fl32(5.1) + fl32(skin)."""
    consts, widths, params, om = model
    n = len(species)
    ctx = U.gpu_create(consts, widths, params, 1, n)
    try:
        U.gpu_energy_forces(ctx, species, xyz, box, skin=skin)
        return U.gpu_neighbors(ctx, 0, n, stride=160)
    finally:
        nnp.nnp_destroy(ctx)


def test_no_alloc_neighbour_lists_equal_the_existing_path_twice_in_a_row():
    model = U.make_model(1)
    rng = np.random.default_rng(5)
    # call 1: 1000 waters, coordinates unwrapped by up to two box lengths; call 2 right after it: another system with fewer
    # atoms and fewer cells (the shared array still holds call 1's positions, order and cursor); call 3: the first again
    sp1, xyz1, box1 = inputs.water_box(1000)
    xyz1 = (xyz1 + rng.integers(-2, 3, size=xyz1.shape) * box1).astype(np.float32).astype(np.float64)
    sp2, xyz2, box2 = inputs.water_box(216, seed=inputs.SEED0 + 17)
    cases = [(sp1, xyz1, box1, 0.3), (sp2, xyz2, box2, 0.0), (sp1, xyz1, box1, 0.3)]
    got = [_rows_no_alloc(xyz, box, float(np.float32(5.1) + np.float32(skin))) for sp, xyz, box, skin in cases]
    for (sp, xyz, box, skin), rows in zip(cases, got):
        want = _rows_existing(model, sp, xyz, box, skin)
        bad = [i for i in range(len(sp)) if not np.array_equal(rows[i], want[i])]
        assert not bad, (len(sp), skin, len(bad), bad[:5])
    assert sum(len(r) for r in got[0]) > 50 * len(sp1)  # (the lists are not trivially empty)


def test_no_alloc_non_periodic_cluster_and_side_stream():
    model = U.make_model(1)
    sp, xyz, box = inputs.water_box(216)
    keep = np.argsort(((xyz - xyz.mean(0)) ** 2).sum(1))[:300]
    sp, xyz = sp[keep].astype(np.int32), xyz[keep]
    st = torch.cuda.Stream()
    rows = _rows_no_alloc(xyz, None, float(np.float32(5.1)), stream=st.cuda_stream)
    want = _rows_existing(model, sp, xyz, None, 0.0)
    assert all(np.array_equal(rows[i], want[i]) for i in range(len(sp)))


def test_no_alloc_rejects_what_does_not_fit():
    dev = torch.device("cuda:0")
    n = nnp.NNP_NO_ALLOC_MAX_ATOMS + 1
    d_x = torch.zeros((n, 3), dtype=torch.float32, device=dev)
    d_c = torch.zeros(n, dtype=torch.int32, device=dev)
    d_l = torch.zeros((n, 4), dtype=torch.int32, device=dev)
    with pytest.raises(nnp.NnpError) as e:
        nnp.nnp_neighbors_no_alloc(n, d_x, [40.0, 40.0, 40.0], 5.1, d_c, d_l, 4)
    assert e.value.status == nnp.NNP_EINVAL and "NNP_NO_ALLOC_MAX_ATOMS" in str(e.value)
    with pytest.raises(nnp.NnpError) as e:  # minimum image not unique
        nnp.nnp_neighbors_no_alloc(8, d_x, [9.0, 40.0, 40.0], 5.1, d_c, d_l, 4)
    assert e.value.status == nnp.NNP_EBOX
    nnp.nnp_neighbors_no_alloc(0, None, None, 5.1, None, None, 4)  # empty: a no-op
