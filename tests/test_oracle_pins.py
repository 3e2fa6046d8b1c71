"""Pins for oracle/ (CPU only).  Each test states which plausible mistake it would catch.

Citations: SURVEY.md 8(c) C1 (O1-O7), C2 (readings), C3 (pins); PAPER.md L41 (directed lists, batching),
L61 (cosine switch, continuity at the cutoff), L176 (Fig. 2 pipeline), L307 (velocity Verlet), L443 (angular form).
"""
import math

import numpy as np
import pytest
from scipy.spatial import cKDTree

from oracle import nnp_oracle as orc
from paper_2405_01491_b200 import inputs


def rot(seed):
    return inputs._random_rotations(np.random.default_rng(seed), 1)[0]


# ---------------------------------------------------------------- sizes / indexing
def test_aev_length_closed_form(ani_model):
    # BASELINE.json: 7x16 radial + 28x4x8 angular = 1008
    assert ani_model.aev_len == 7 * 16 + 28 * 4 * 8 == 1008


def test_pair_index_is_upper_triangle_bijection():
    seen = {}
    for s in range(7):
        for t in range(s, 7):
            p = orc.pair_index(7, s, t)
            assert orc.pair_index(7, t, s) == p
            seen[p] = (s, t)
    assert sorted(seen) == list(range(28))
    assert orc.pair_index(7, 6, 6) == 27 and orc.pair_index(7, 0, 0) == 0 and orc.pair_index(7, 1, 1) == 7
    # row-major: p increases with t inside a row, rows in order of s
    order = [seen[p] for p in range(28)]
    assert order == sorted(order)


# ---------------------------------------------------------------- scalar pieces: values known without the formula
def test_cutoff_function_special_values():
    R = 5.1
    assert orc.fc(0.0, R) == 1.0
    assert abs(orc.fc(R / 2, R) - 0.5) < 1e-15
    assert abs(orc.fc(R / 3, R) - 0.75) < 1e-15          # cos(pi/3) = 1/2
    assert orc.fc(R, R) == 0.0 and orc.fc(R * 1.0001, R) == 0.0 and orc.fc(2 * R, R) == 0.0   # reading A4
    assert 0 < orc.fc(R * (1 - 1e-6), R) < 1e-11          # goes smoothly to zero


def test_celu_special_values():
    a = 0.1
    assert orc.celu(0.0, a) == 0.0
    assert orc.celu(2.5, a) == 2.5
    assert abs(orc.celu(-50.0, a) + a) < 1e-15
    assert abs(orc.celu(-a * math.log(2.0), a) + a / 2) < 1e-15      # alpha(e^{-ln2}-1) = -alpha/2


# ---------------------------------------------------------------- radial block
def test_isolated_atom_and_beyond_cutoff_zero(ani_model):
    r = orc.energy_forces(ani_model, [3], [[0, 0, 0]], want_aev=True)
    assert np.all(r["aev"] == 0)
    r = orc.energy_forces(ani_model, [3, 0], [[0, 0, 0], [5.1, 0, 0]], want_aev=True)
    assert np.all(r["aev"] == 0) and np.all(r["F"] == 0)


def test_dimer_radial_hand_values(ani_model, consts):
    # r = ShfR_k exactly => Gaussian = 1 => G[s_j*16+k] = fc(r)/4 ; and at r = R/2, fc = 1/2.
    for k in (0, 5, 15):
        r0 = float(consts["shf_r"][k])
        res = orc.energy_forces(ani_model, [3, 1], [[0, 0, 0], [0, r0, 0]], want_aev=True)
        G = res["aev"]
        # atom 0 (O) sees a C (species 1): block 1; atom 1 sees an O (species 3): block 3
        assert abs(G[0, 1 * 16 + k] - 0.25 * (0.5 * math.cos(math.pi * r0 / 5.1) + 0.5)) < 1e-15
        assert abs(G[1, 3 * 16 + k] - G[0, 1 * 16 + k]) < 1e-16
        nz = np.nonzero(G[0])[0]
        assert nz.min() >= 16 and nz.max() < 32           # only the neighbour-species block, no angular terms
        # neighbouring shifts: ratio exp(-eta*Delta^2) with Delta = 0.26875
        if k < 15:
            assert abs(G[0, 16 + k + 1] / G[0, 16 + k] - math.exp(-19.7 * 0.26875 ** 2)) < 1e-12
    res = orc.energy_forces(ani_model, [0, 0], [[1, 1, 1], [1, 1, 1 + 2.55]], want_aev=True)
    k = 7   # shf_r[7] = 2.68125
    assert abs(res["aev"][0, k] - 0.125 * math.exp(-19.7 * (2.55 - 2.68125) ** 2)) < 1e-15


def test_radial_additivity_over_neighbours(ani_model):
    # two neighbours of the same species beyond the angular cutoff of each other's pairing: radial block adds
    a = orc.energy_forces(ani_model, [0, 3], [[0, 0, 0], [4.0, 0, 0]], want_aev=True)["aev"][0]
    b = orc.energy_forces(ani_model, [0, 3], [[0, 0, 0], [0, 4.5, 0]], want_aev=True)["aev"][0]
    c = orc.energy_forces(ani_model, [0, 3, 3], [[0, 0, 0], [4.0, 0, 0], [0, 4.5, 0]], want_aev=True)["aev"][0]
    assert np.allclose(c, a + b, atol=1e-16)
    assert np.all(c[112:] == 0)       # both beyond 3.5 A: no angular term


# ---------------------------------------------------------------- angular block
def _trimer(r, theta, sj=0, sk=0, si=3):
    xyz = [[0, 0, 0], [r, 0, 0], [r * math.cos(theta), r * math.sin(theta), 0]]
    return [si, sj, sk], xyz


def test_trimer_angular_hand_values(ani_model, consts):
    # r_ij = r_ik = ShfA_a and 0.95 cos(theta) = cos(ShfZ_z)  =>  both factors are exactly 1
    # => G[112 + p*32 + a*4 + z] = 2 fc(r)^2
    for a in (0, 3, 7):
        for z in (0, 1, 2, 3):
            r = float(consts["shf_a"][a])
            theta = math.acos(math.cos(float(consts["shf_z"][z])) / 0.95)
            sp, xyz = _trimer(r, theta, 0, 0)
            G = orc.energy_forces(ani_model, sp, xyz, want_aev=True)["aev"][0]
            fcv = 0.5 * math.cos(math.pi * r / 3.5) + 0.5
            p = 0   # (H,H)
            assert abs(G[112 + p * 32 + a * 4 + z] - 2 * fcv * fcv) < 1e-13
            assert np.all(G[112 + 32:] == 0)              # nothing outside block (H,H)


def test_trimer_angular_off_peak_values(ani_model, consts):
    """The angular term AWAY from its peaks (the form ((1+cos(theta'-ShfZ))/2)^zeta is PAPER.md L443).
    Each case makes all but one factor exactly 1, so the remaining factor has a value known without the formula:
    (i) pins the zeta power, (ii) pins eta_A and that r-bar is the ARITHMETIC mean, (iii) pins the ShfA spacing."""
    eta_a, zeta = float(consts["eta_a"]), float(consts["zeta"])
    shf_a, shf_z = np.asarray(consts["shf_a"], float), np.asarray(consts["shf_z"], float)
    fc = lambda r: 0.5 * math.cos(math.pi * r / 3.5) + 0.5          # noqa: E731  pinned by test_cutoff_function_special_values
    # (i) theta' = ShfZ_z +- pi/2  =>  (1 + cos(+-pi/2))/2 = 1/2  =>  G = 2 * 2^-zeta * fc^2  at r_ij = r_ik = ShfA_a
    for z, sign in ((0, +1), (1, +1), (2, -1), (3, -1)):
        thp = shf_z[z] + sign * math.pi / 2                          # inside [acos(.95), acos(-.95)] for these four
        theta = math.acos(math.cos(thp) / 0.95)
        for a in (1, 4):
            r = float(shf_a[a])
            sp, xyz = _trimer(r, theta)
            G = orc.energy_forces(ani_model, sp, xyz, want_aev=True)["aev"][0]
            want = 2.0 * 2.0 ** (-zeta) * fc(r) ** 2
            assert abs(G[112 + a * 4 + z] / want - 1.0) < 1e-11, (z, a, G[112 + a * 4 + z], want)
    # (ii) on-peak angle, r_ik = ShfA_a, r_ij = ShfA_a + 2 delta  =>  r-bar = ShfA_a + delta (arithmetic mean; the geometric
    #      mean sqrt(s (s + 2 delta)) differs in the 2nd digit of the exponent)  =>  G = 2 exp(-eta_A delta^2) fc(r_ij) fc(r_ik)
    for a, delta in ((2, 0.11), (5, -0.17), (0, 0.3)):
        for z in (0, 2):
            s = float(shf_a[a])
            theta = math.acos(math.cos(shf_z[z]) / 0.95)
            rj, rk = s + 2 * delta, s
            xyz = [[0, 0, 0], [rj, 0, 0], [rk * math.cos(theta), rk * math.sin(theta), 0]]
            G = orc.energy_forces(ani_model, [3, 0, 0], xyz, want_aev=True)["aev"][0]
            want = 2.0 * math.exp(-eta_a * delta * delta) * fc(rj) * fc(rk)
            assert abs(G[112 + a * 4 + z] / want - 1.0) < 1e-11, (a, z, G[112 + a * 4 + z], want)
            geo = 2.0 * math.exp(-eta_a * (math.sqrt(rj * rk) - s) ** 2) * fc(rj) * fc(rk)
            assert abs(geo / want - 1.0) > 1e-4                       # the case does tell the two means apart
    # (iii) r_ij = r_ik = ShfA_a at the on-peak angle: feature a+1 / feature a = exp(-eta_A Delta^2), Delta = 0.3375;
    #       two shifts on: exp(-4 eta_A Delta^2)
    dlt = 0.3375
    for a in (0, 3, 5):
        theta = math.acos(math.cos(shf_z[1]) / 0.95)
        sp, xyz = _trimer(float(shf_a[a]), theta)
        G = orc.energy_forces(ani_model, sp, xyz, want_aev=True)["aev"][0]
        assert abs(G[112 + (a + 1) * 4 + 1] / G[112 + a * 4 + 1] / math.exp(-eta_a * dlt ** 2) - 1.0) < 1e-11
        assert abs(G[112 + (a + 2) * 4 + 1] / G[112 + a * 4 + 1] / math.exp(-4 * eta_a * dlt ** 2) - 1.0) < 1e-11
    # and between neighbouring ShfZ at theta' = (ShfZ_0 + ShfZ_1)/2: equal bases => equal features (symmetric about the midpoint)
    thp = 0.5 * (shf_z[0] + shf_z[1])
    sp, xyz = _trimer(1.9, math.acos(math.cos(thp) / 0.95))
    G = orc.energy_forces(ani_model, sp, xyz, want_aev=True)["aev"][0]
    assert abs(G[112 + 3 * 4 + 0] / G[112 + 3 * 4 + 1] - 1.0) < 1e-11
    # value there: base = (1 + cos(pi/8))/2 = cos^2(pi/16)
    want = 2.0 * math.cos(math.pi / 16) ** (2 * zeta) * math.exp(-eta_a * (1.9 - shf_a[3]) ** 2) * fc(1.9) ** 2
    assert abs(G[112 + 3 * 4 + 0] / want - 1.0) < 1e-11


def test_trimer_block_placement_and_swap(ani_model):
    r, th = 1.7, 1.9
    for sj, sk in ((0, 3), (1, 6), (6, 6), (2, 4)):
        sp, xyz = _trimer(r, th, sj, sk)
        G = orc.energy_forces(ani_model, sp, xyz, want_aev=True)["aev"][0]
        p = orc.pair_index(7, sj, sk)
        ang = G[112:].reshape(28, 32)
        assert np.all(ang[p] > 0)
        assert np.all(np.delete(ang, p, axis=0) == 0)
        sp2, xyz2 = [sp[0], sp[2], sp[1]], [xyz[0], xyz[2], xyz[1]]      # swap j and k
        G2 = orc.energy_forces(ani_model, sp2, xyz2, want_aev=True)["aev"][0]
        assert np.allclose(G, G2, rtol=0, atol=1e-16)


def test_trimer_collinear_angles_finite(ani_model):
    for th in (0.0 + 1e-9, math.pi / 2, math.pi):
        sp, xyz = _trimer(1.5, th)
        xyz[2] = [1.2 * math.cos(th), 1.2 * math.sin(th), 0.0]
        res = orc.energy_forces(ani_model, sp, xyz, want_aev=True)
        assert np.all(np.isfinite(res["aev"])) and np.all(np.isfinite(res["F"]))


def test_angular_uses_angular_cutoff_only(ani_model):
    # k at 3.6 A (> 3.5): contributes radially, but no triplet
    sp, xyz = [3, 0, 0], [[0, 0, 0], [1.0, 0, 0], [0, 3.6, 0]]
    G = orc.energy_forces(ani_model, sp, xyz, want_aev=True)["aev"][0]
    assert np.all(G[112:] == 0) and G[:16].sum() > 0
    xyz[2] = [0, 3.4, 0]
    G = orc.energy_forces(ani_model, sp, xyz, want_aev=True)["aev"][0]
    assert G[112:144].sum() > 0


# ---------------------------------------------------------------- MLP vs library routines
def _numpy_mlp(widths_row, params_iter, G, alpha=0.1):
    h = G
    nl = len(widths_row) - 1
    Ws = []
    for l in range(nl):
        fi, fo = widths_row[l], widths_row[l + 1]
        W = next(params_iter)(fi * fo).reshape(fi, fo)
        b = next(params_iter)(fo)
        Ws.append((W, b))
    zs = []
    for l, (W, b) in enumerate(Ws):
        z = h @ W + b
        zs.append(z)
        h = np.where(z > 0, z, alpha * np.expm1(z / alpha)) if l < nl - 1 else z
    # reverse mode by hand with numpy
    d = np.ones(1)
    for l in range(nl - 1, -1, -1):
        W, _ = Ws[l]
        d = W @ d
        if l > 0:
            d = d * np.where(zs[l - 1] > 0, 1.0, np.exp(zs[l - 1] / alpha))
    return h[0], d


def test_mlp_matches_numpy_matmul_all_species(consts):
    p = inputs.make_weights(7, 2, bias_std=0.3)
    m = orc.OracleModel(consts, inputs.WIDTHS, p, 2)
    rng = np.random.default_rng(0)
    pos = [0]

    def taker():
        while True:
            def take(n):
                out = p[pos[0]:pos[0] + n]
                pos[0] += n
                return out
            yield take
    it = taker()
    for net in range(2):
        for s in range(7):
            G = rng.normal(size=1008) * 0.5
            e_ref, g_ref = _numpy_mlp(list(inputs.WIDTHS[s]), it, G)
            e, g = m.mlp(net, s, G, want_grad=True)
            assert abs(e - e_ref) < 1e-12 * max(1, abs(e_ref))
            assert np.allclose(g, g_ref, rtol=1e-11, atol=1e-13)
    assert pos[0] == p.size


def test_mlp_zero_weights_gives_bias_chain_and_single_layer_dot(consts):
    w = np.array([[1008, 1]] * 7, dtype=np.int32)
    rng = np.random.default_rng(1)
    p = rng.normal(size=7 * 1009)
    m = orc.OracleModel(consts, w, p, 1)
    G = rng.normal(size=1008)
    for s in range(7):
        W, b = p[s * 1009:s * 1009 + 1008], p[s * 1009 + 1008]
        e, g = m.mlp(0, s, G, want_grad=True)
        assert abs(e - (G @ W + b)) < 1e-12 and np.allclose(g, W)
    w2 = np.array([[1008, 4, 1]] * 7, dtype=np.int32)
    p2 = np.zeros(7 * (1008 * 4 + 4 + 4 + 1))
    per = 1008 * 4 + 4 + 4 + 1
    p2[1008 * 4:1008 * 4 + 4] = [-1.0, 0.5, 0.0, -0.05]       # b1
    p2[1008 * 4 + 4:1008 * 4 + 8] = [1.0, 2.0, 3.0, 4.0]      # W2
    p2[per - 1] = 0.25
    m2 = orc.OracleModel(consts, w2, p2, 1)
    expect = 0.1 * math.expm1(-10.0) * 1 + 0.5 * 2 + 0 + 0.1 * math.expm1(-0.5) * 4 + 0.25
    assert abs(m2.mlp(0, 0, G) - expect) < 1e-14


# ---------------------------------------------------------------- neighbours
def _kdtree_sets(xyz, box, r, mol_id=None):
    if box is not None:
        t = cKDTree(np.mod(xyz, box), boxsize=box)
        rows = t.query_ball_point(np.mod(xyz, box), r)
    else:
        t = cKDTree(xyz)
        rows = t.query_ball_point(xyz, r)
    out = []
    for i, row in enumerate(rows):
        out.append(sorted(j for j in row if j != i and (mol_id is None or mol_id[j] == mol_id[i])))
    return out


def test_brute_force_neighbours_vs_kdtree_periodic(water64):
    sp, xyz, box = water64
    for r in (3.5, 5.1, 5.6):
        mine = orc.neighbors(xyz, box, r)
        ref = _kdtree_sets(xyz, box, r * (1 - 1e-12))
        assert all(list(a) == b for a, b in zip(mine, ref))
        # directed list: j in N(i) <=> i in N(j)
        S = [set(a.tolist()) for a in mine]
        assert all(i in S[j] for i in range(len(S)) for j in S[i])


def test_neighbour_counts_match_density(consts):
    sp, xyz, box = inputs.water_box(512, seed=3)
    rho = len(sp) / box[0] ** 3
    for r, expect in ((5.1, 55.7), (3.5, 18.0)):
        c = np.mean([len(a) for a in orc.neighbors(xyz, box, r, method="grid")])
        assert abs(c - rho * 4 / 3 * math.pi * r ** 3) / c < 0.08
        assert abs(c - expect) / expect < 0.08          # SURVEY 8(a) figures for water


def test_grid_neighbours_equal_brute_force():
    sp, xyz, box = inputs.water_box(300, seed=5)
    xyz = xyz + np.random.default_rng(0).integers(-2, 3, size=xyz.shape) * box     # unwrapped coordinates too
    for r in (3.5, 5.6):
        for f32 in (False, True):
            a = orc.neighbors(xyz, box, r, fp32_pred=f32, method="brute")
            b = orc.neighbors(xyz, box, r, fp32_pred=f32, method="grid")
            assert all(np.array_equal(x, y) for x, y in zip(a, b))


def test_fp32_predicate_agrees_outside_guard_band(water64):
    sp, xyz, box = water64
    r = 5.6
    a = orc.neighbors(xyz, box, r, fp32_pred=True)
    lo = orc.neighbors(xyz, box, r - 1e-4)
    hi = orc.neighbors(xyz, box, r + 1e-4)
    for x, l, h in zip(a, lo, hi):
        assert set(l.tolist()) <= set(x.tolist()) <= set(h.tolist())


def test_molecule_batch_never_pairs_across_molecules():
    sp, xyz, offs = inputs.molecule_batch(6, seed=2)
    xyz = xyz.copy()
    xyz[offs[1]:offs[2]] += xyz[0] - xyz[offs[1]]       # put molecule 1 on top of molecule 0
    mol = np.repeat(np.arange(6), np.diff(offs)).astype(np.int32)
    rows = orc.neighbors(xyz, None, 5.1, mol_id=mol)
    assert all(mol[j] == mol[i] for i, row in enumerate(rows) for j in row)
    assert [list(r) for r in rows] == _kdtree_sets(xyz, None, 5.1, mol)


# ---------------------------------------------------------------- forces: finite differences and invariances
def _fd_check(model, sp, xyz, box, idx, h=1e-4, mol_offsets=None):
    base = orc.energy_forces(model, sp, xyz, box, mol_offsets)
    err = 0.0
    for (i, c) in idx:
        xp, xm = np.array(xyz), np.array(xyz)
        xp[i, c] += h
        xm[i, c] -= h
        ep = orc.energy_forces(model, sp, xp, box, mol_offsets, want_forces=False)["E"].sum()
        em = orc.energy_forces(model, sp, xm, box, mol_offsets, want_forces=False)["E"].sum()
        fd = -(ep - em) / (2 * h)
        err = max(err, abs(fd - base["F"][i, c]))
    return err, np.abs(base["F"]).max()


def test_forces_equal_minus_gradient_periodic_water_small_model(small_model, water64):
    sp, xyz, box = water64
    rng = np.random.default_rng(0)
    idx = [(int(rng.integers(192)), int(rng.integers(3))) for _ in range(40)]
    err, fmax = _fd_check(small_model, sp, xyz, box, idx)
    assert fmax > 1e-3 and err < 2e-7 * max(1.0, fmax)


def test_forces_equal_minus_gradient_ani_widths(ani_model, water64):
    sp, xyz, box = water64
    idx = [(0, 0), (1, 2), (100, 1), (191, 0)]
    err, fmax = _fd_check(ani_model, sp, xyz, box, idx)
    assert fmax > 1e-3 and err < 2e-7 * max(1.0, fmax)


def test_forces_equal_minus_gradient_all_species_molecule(small_model):
    sp, xyz, offs = inputs.molecule_batch(3, nmin=12, nmax=14, seed=11)
    sp = (np.arange(len(sp)) % 7).astype(np.int32)       # every species and every species pair present
    idx = [(i, c) for i in range(0, len(sp), 3) for c in range(3)]
    err, fmax = _fd_check(small_model, sp, xyz, None, idx, mol_offsets=offs)
    assert fmax > 1e-3 and err < 2e-7 * max(1.0, fmax)


def test_net_force_and_torque_vanish(small_model, water64):
    sp, xyz, box = water64
    F = orc.energy_forces(small_model, sp, xyz, box)["F"]
    assert np.abs(F.sum(0)).max() < 1e-10 * np.abs(F).sum()
    sp, xyz, offs = inputs.molecule_batch(2, seed=4)
    r = orc.energy_forces(small_model, sp, xyz, None, offs)
    for m in range(2):
        sl = slice(offs[m], offs[m + 1])
        assert np.abs(r["F"][sl].sum(0)).max() < 1e-11
        assert np.abs(np.cross(xyz[sl], r["F"][sl]).sum(0)).max() < 1e-10


def test_rotation_translation_invariance_nonperiodic(small_model):
    sp, xyz, offs = inputs.molecule_batch(1, nmin=20, nmax=20, seed=9)
    a = orc.energy_forces(small_model, sp, xyz)
    R = rot(1)
    b = orc.energy_forces(small_model, sp, xyz @ R.T + np.array([3.0, -2.0, 0.7]))
    assert abs(a["E"][0] - b["E"][0]) < 1e-11 * max(1, abs(a["E"][0]))
    assert np.allclose(a["F"] @ R.T, b["F"], atol=1e-10)


def test_periodic_symmetries(small_model, water64):
    sp, xyz, box = water64
    a = orc.energy_forces(small_model, sp, xyz, box)
    # cubic symmetry: x->y->z->x and a mirror
    P = np.array([[0, 1, 0], [0, 0, 1], [1, 0, 0]], dtype=float)
    b = orc.energy_forces(small_model, sp, xyz @ P.T, box)
    assert abs(a["E"][0] - b["E"][0]) < 1e-10 and np.allclose(a["F"] @ P.T, b["F"], atol=1e-10)
    M = np.diag([1.0, -1.0, 1.0])
    b = orc.energy_forces(small_model, sp, xyz @ M, box)
    assert abs(a["E"][0] - b["E"][0]) < 1e-10 and np.allclose(a["F"] @ M, b["F"], atol=1e-10)
    # global translation, and wrapping individual atoms by lattice vectors
    b = orc.energy_forces(small_model, sp, xyz + np.array([1.234, -7.0, 30.1]), box)
    assert abs(a["E"][0] - b["E"][0]) < 1e-9 and np.allclose(a["F"], b["F"], atol=1e-9)
    sh = np.random.default_rng(0).integers(-2, 3, size=xyz.shape) * box
    b = orc.energy_forces(small_model, sp, xyz + sh, box)
    assert abs(a["E"][0] - b["E"][0]) < 1e-9 and np.allclose(a["F"], b["F"], atol=1e-9)


def test_same_species_permutation_invariance(small_model, water64):
    sp, xyz, box = water64
    a = orc.energy_forces(small_model, sp, xyz, box)
    perm = np.random.default_rng(2).permutation(len(sp))
    b = orc.energy_forces(small_model, sp[perm], xyz[perm], box)
    assert abs(a["E"][0] - b["E"][0]) < 1e-10
    assert np.allclose(a["F"][perm], b["F"], atol=1e-11)
    # swapping two atoms' species labels of different species must change the energy
    sp2 = sp.copy()
    sp2[0], sp2[1] = sp[1], sp[0]
    assert abs(orc.energy_forces(small_model, sp2, xyz, box)["E"][0] - a["E"][0]) > 1e-6


def test_energy_and_force_continuous_across_cutoffs(small_model):
    # no discontinuity when atoms enter/leave the neighbourhood
    base = [[0, 0, 0], [1.0, 0.2, 0], [-0.3, 1.1, 0.4]]
    sp = [3, 0, 0, 1]
    for R in (5.1, 3.5):
        vals = []
        for dr in (-1e-7, 1e-7):
            xyz = base + [[0.0, 0.0, R + dr]]
            r = orc.energy_forces(small_model, sp, xyz)
            vals.append((r["E"][0], r["F"].copy()))
        assert abs(vals[0][0] - vals[1][0]) < 1e-9
        assert np.abs(vals[0][1] - vals[1][1]).max() < 1e-5


def test_extensivity_under_box_replication(small_model, water64):
    sp, xyz, box = water64
    a = orc.energy_forces(small_model, sp, xyz, box)
    sp2, xyz2, box2 = inputs.replicate(sp, xyz, box, 2)
    b = orc.energy_forces(small_model, sp2, xyz2, box2, nbr_method=1)
    assert abs(b["E"][0] - 8 * a["E"][0]) < 1e-9 * abs(a["E"][0]) * 8 + 1e-9
    assert np.allclose(b["F"].reshape(8, -1, 3), a["F"][None], atol=1e-10)
    c = orc.energy_forces(small_model, sp2, xyz2, box2, nbr_method=0)
    assert np.allclose(b["F"], c["F"], atol=1e-12) and abs(b["E"][0] - c["E"][0]) < 1e-9


def test_ensemble_identities(consts, small_widths, water64):
    sp, xyz, box = water64
    p = inputs.make_weights(21, 3, widths=small_widths, bias_std=0.2)
    per = p.size // 3
    singles = [orc.energy_forces(orc.OracleModel(consts, small_widths, p[k * per:(k + 1) * per], 1), sp, xyz, box)
               for k in range(3)]
    ens = orc.energy_forces(orc.OracleModel(consts, small_widths, p, 3), sp, xyz, box)
    assert abs(ens["E"][0] - np.mean([s["E"][0] for s in singles])) < 1e-10           # reading B5: mean
    assert np.allclose(ens["F"], np.mean([s["F"] for s in singles], axis=0), atol=1e-12)
    same = orc.energy_forces(orc.OracleModel(consts, small_widths, np.tile(p[:per], 8), 8), sp, xyz, box)
    assert abs(same["E"][0] - singles[0]["E"][0]) < 1e-10 and np.allclose(same["F"], singles[0]["F"], atol=1e-12)


def test_batch_equals_each_molecule_alone(small_model):
    sp, xyz, offs = inputs.molecule_batch(5, seed=6)
    xyz = xyz.copy()
    xyz[offs[2]:offs[3]] += xyz[offs[1]] - xyz[offs[2]]      # overlapping molecules must still not interact
    b = orc.energy_forces(small_model, sp, xyz, None, offs)
    for m in range(5):
        sl = slice(offs[m], offs[m + 1])
        a = orc.energy_forces(small_model, sp[sl], xyz[sl])
        assert abs(a["E"][0] - b["E"][m]) < 1e-11 and np.allclose(a["F"], b["F"][sl], atol=1e-12)


def test_periodic_replica_batch_equals_each_replica_alone(small_model, water64):
    """Replicas of one periodic cell (the beads of a ring polymer; L41: same batch index => edge): the
    batched energies and forces are those of each replica run alone in the same box."""
    sp1, x1, box = water64
    rng = np.random.default_rng(77)
    reps = [x1 + 0.05 * rng.standard_normal(x1.shape) * (r > 0) for r in range(3)]
    sp = np.tile(sp1, 3)
    xyz = np.concatenate(reps)
    offs = np.arange(4, dtype=np.int32) * len(sp1)
    b = orc.energy_forces(small_model, sp, xyz, box, offs)
    for r in range(3):
        a = orc.energy_forces(small_model, sp1, reps[r], box)
        assert abs(a["E"][0] - b["E"][r]) < 1e-10 and np.allclose(a["F"], b["F"][offs[r]:offs[r + 1]], atol=1e-11)
    assert abs(b["E"][1] - b["E"][0]) > 1e-6   # the replicas do differ


def test_self_energy_shifts_energy_only(consts, small_widths, water64):
    sp, xyz, box = water64
    p = inputs.make_weights(5, 1, widths=small_widths)
    se = np.arange(7) * 1.5 - 2.0
    a = orc.energy_forces(orc.OracleModel(consts, small_widths, p, 1), sp, xyz, box)
    b = orc.energy_forces(orc.OracleModel(consts, small_widths, p, 1, self_energy=se), sp, xyz, box)
    assert abs(b["E"][0] - a["E"][0] - se[sp].sum()) < 1e-9 and np.allclose(a["F"], b["F"], rtol=0, atol=1e-13)


# ---------------------------------------------------------------- MD (O7)
def _md_setup(small_model):
    sp, xyz, box = inputs.water_box(27, seed=8)
    v = inputs.maxwell_boltzmann(sp, 300.0, seed=1)
    return sp, xyz, box, v


def test_velocity_verlet_time_reversible(small_model):
    sp, xyz, box, v = _md_setup(small_model)
    a = orc.md(small_model, sp, xyz, v, inputs.MASS, box, 0.5, inputs.ACCEL_CONV, 20)
    b = orc.md(small_model, sp, a["xyz"], -a["vel"], inputs.MASS, box, 0.5, inputs.ACCEL_CONV, 20)
    assert np.abs(b["xyz"] - xyz).max() < 1e-10 and np.abs(b["vel"] + v).max() < 1e-11


def test_velocity_verlet_energy_error_scales_dt2(small_model):
    sp, xyz, box, v = _md_setup(small_model)
    errs = []
    for dt, n in ((0.5, 40), (0.25, 80)):
        r = orc.md(small_model, sp, xyz, v, inputs.MASS, box, dt, inputs.ACCEL_CONV, n)
        tot = r["epot"] + r["ekin"]
        errs.append(np.abs(tot - tot[0]).max())
    assert errs[0] > 0 and 2.5 < errs[0] / errs[1] < 6.0


def test_velocity_verlet_first_step_by_hand(small_model):
    sp, xyz, box, v = _md_setup(small_model)
    dt = 0.5
    F0 = orc.energy_forces(small_model, sp, xyz, box)["F"]
    a0 = inputs.ACCEL_CONV * F0 / inputs.MASS[sp][:, None]
    x1 = xyz + dt * v + 0.5 * dt * dt * a0                       # textbook velocity-Verlet position update
    F1 = orc.energy_forces(small_model, sp, x1, box)["F"]
    v1 = v + 0.5 * dt * (a0 + inputs.ACCEL_CONV * F1 / inputs.MASS[sp][:, None])
    r = orc.md(small_model, sp, xyz, v, inputs.MASS, box, dt, inputs.ACCEL_CONV, 1)
    assert np.abs(r["xyz"] - x1).max() < 1e-13 and np.abs(r["vel"] - v1).max() < 1e-14
    ke = 0.5 * (inputs.MASS[sp][:, None] * v ** 2).sum() / inputs.ACCEL_CONV
    assert abs(r["ekin"][0] - ke) < 1e-10
    # kinetic temperature of the seeded Maxwell-Boltzmann draw is near 300 K (reading C3)
    T = 2 * ke / (3 * len(sp) * inputs.KB)
    assert 200 < T < 400


def test_rebuild_rule_strict_half_skin():
    x0 = np.zeros((4, 3))
    x1 = x0.copy()
    x1[2, 1] = 0.25
    assert not orc.needs_rebuild(x1, x0, 0.5)          # == skin/2: strict (reading C2)
    x1[2, 1] = 0.2500001
    assert orc.needs_rebuild(x1, x0, 0.5)
    x1[2] = [0.15, 0.15, 0.15]                          # |d| = 0.2598 > 0.25
    assert orc.needs_rebuild(x1, x0, 0.5)


def test_md_rebuild_count_reasonable(small_model):
    sp, xyz, box, v = _md_setup(small_model)
    r = orc.md(small_model, sp, xyz, v, inputs.MASS, box, 0.5, inputs.ACCEL_CONV, 30, skin=0.5)
    assert 2 <= r["n_rebuilds"] <= 12


# ---------------------------------------------------------------- regression pin (values written by tests/golden/make_oracle_golden.py)
def test_oracle_matches_stored_golden(consts):
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "oracle_water64.txt")
    params = inputs.make_weights(inputs.SEED0, 1, last_layer_scale=inputs.FORCE_SCALE_WATER, bias_std=0.05)
    om = orc.OracleModel(consts, inputs.WIDTHS, params, 1)
    sp, xyz, box = inputs.water_box(64, 12.42)
    r = orc.energy_forces(om, sp, xyz, box, want_aev=True)
    for line in open(path):
        t = line.split()
        if t[0] == "E":
            assert abs(r["E"][0] - float(t[1])) < 1e-9 * abs(float(t[1]))
        elif t[0] == "F":
            assert np.allclose(r["F"][int(t[1])], [float(x) for x in t[2:5]], rtol=1e-9, atol=1e-9)
        elif t[0] == "AEVSUM":
            assert abs(r["aev"].sum() - float(t[1])) < 1e-9 * float(t[1])
        elif t[0] == "AEVNNZ":
            # water: only H,O radial blocks and the (H,H),(H,O),(O,O) angular blocks can be non-zero
            assert int((r["aev"] != 0).sum()) == int(t[1]) <= 192 * 128


# ---------------------------------------------------------------- NEXT-1: Langevin BAOAB
def test_philox4x32_10_known_answers():
    """Known-answer vectors of Philox4x32-10 from the reference distribution of Salmon et al. (SC'11), kat_vectors:
    zero counter/key, all-ones counter/key, and the digits-of-pi counter/key."""
    assert orc.philox4x32_10([0, 0, 0, 0], [0, 0]) == [0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8]
    assert orc.philox4x32_10([0xffffffff] * 4, [0xffffffff] * 2) == [0x408f276d, 0x41c83b0e, 0xa20bc7c6, 0x6d5451fd]
    assert orc.philox4x32_10([0x243f6a88, 0x85a308d3, 0x13198a2e, 0x03707344], [0xa4093822, 0x299f31d0]) == \
        [0xd16cfe09, 0x94fdcceb, 0x5001e420, 0x24126ea1]


def test_langevin_normals_are_standard_normal():
    from scipy import stats
    xi = np.array([orc.langevin_normals(a, s, 20240501) for a in range(400) for s in range(25)])
    assert xi.shape == (10000, 3)
    for c in range(3):
        assert stats.kstest(xi[:, c], "norm").pvalue > 1e-3
    assert np.abs(xi.mean(0)).max() < 0.04 and np.abs(xi.var(0) - 1).max() < 0.05
    assert np.abs(np.corrcoef(xi.T) - np.eye(3)).max() < 0.04
    # different atoms, steps and seeds give different numbers; the same triple repeats
    assert np.array_equal(orc.langevin_normals(5, 9, 1), orc.langevin_normals(5, 9, 1))
    assert not np.array_equal(orc.langevin_normals(5, 9, 1), orc.langevin_normals(5, 9, 2))
    assert not np.array_equal(orc.langevin_normals(5, 9, 1), orc.langevin_normals(6, 9, 1))
    assert not np.array_equal(orc.langevin_normals(5, 9, 1), orc.langevin_normals(5, 10, 1))


def test_langevin_zero_friction_is_velocity_verlet(small_model):
    sp, xyz, box, v = _md_setup(small_model)
    a = orc.md(small_model, sp, xyz, v, inputs.MASS, box, 0.5, inputs.ACCEL_CONV, 12)
    b = orc.md_langevin(small_model, sp, xyz, v, inputs.MASS, box, 0.5, inputs.ACCEL_CONV, 12, gamma=0.0,
                        kT=inputs.KB * 300.0, seed=3)
    assert np.abs(a["xyz"] - b["xyz"]).max() < 1e-12 and np.abs(a["vel"] - b["vel"]).max() < 1e-13
    assert np.abs(a["epot"] - b["epot"]).max() < 1e-9 * np.abs(a["epot"]).max()


def test_langevin_first_step_by_hand(small_model):
    """B A O A (forces) B written out with numpy, the normals taken from the generator."""
    sp, xyz, box, v = _md_setup(small_model)
    dt, gamma, kT, seed, step0 = 0.5, 0.05, inputs.KB * 300.0, 77, 5
    m = inputs.MASS[sp][:, None]
    a0 = inputs.ACCEL_CONV * orc.energy_forces(small_model, sp, xyz, box)["F"] / m
    xi = np.array([orc.langevin_normals(i, step0, seed) for i in range(len(sp))])
    c1 = math.exp(-gamma * dt)
    vb = v + 0.5 * dt * a0
    xa = xyz + 0.5 * dt * vb
    vo = c1 * vb + np.sqrt((1 - c1 * c1) * kT * inputs.ACCEL_CONV / m) * xi
    x1 = xa + 0.5 * dt * vo
    v1 = vo + 0.5 * dt * inputs.ACCEL_CONV * orc.energy_forces(small_model, sp, x1, box)["F"] / m
    r = orc.md_langevin(small_model, sp, xyz, v, inputs.MASS, box, dt, inputs.ACCEL_CONV, 1, gamma, kT, seed, step0=step0)
    assert np.abs(r["xyz"] - x1).max() < 1e-13 and np.abs(r["vel"] - v1).max() < 1e-13
    # the noise really entered: the result differs from the frictionless step by about c2 * |xi|
    r0 = orc.md(small_model, sp, xyz, v, inputs.MASS, box, dt, inputs.ACCEL_CONV, 1)
    assert np.abs(r["vel"] - r0["vel"]).max() > 1e-4


def test_langevin_equipartition_free_particles(small_model):
    """Atoms far apart (no neighbours, zero forces): the O step alone must hold <m v^2> = kT per degree of freedom,
    whatever the start (here: at rest)."""
    n = 64
    sp = (np.arange(n) % 2 * 3).astype(np.int32)                 # H and O
    xyz = 50.0 * np.stack(np.meshgrid(np.arange(4), np.arange(4), np.arange(4), indexing="ij"), -1).reshape(-1, 3).astype(float)
    v = np.zeros((n, 3))
    T = 300.0
    r = orc.md_langevin(small_model, sp, xyz, v, inputs.MASS, None, 0.5, inputs.ACCEL_CONV, 3000, gamma=0.02,
                        kT=inputs.KB * T, seed=11)
    temp = 2 * r["ekin"][500:] / (3 * n * inputs.KB)             # after 5 relaxation times
    assert abs(temp.mean() - T) < 0.06 * T
    assert r["ekin"][0] == 0.0 and np.abs(r["epot"] - r["epot"][0]).max() < 1e-9


# ---------------------------------------------------------------- NEXT-2: virial (PAPER.md L262 energy_and_forces_and_virial)
def test_virial_is_the_strain_derivative_periodic(small_model, water64):
    """V_aa = dE/d eps_aa by central differences of the energy under a homogeneous stretch of coordinates AND box."""
    sp, xyz, box = water64
    r = orc.energy_forces_virial(small_model, sp, xyz, box)
    V, h = r["virial"], 2e-5
    for a in range(3):
        s = np.ones(3)
        s[a] += h
        ep = orc.energy_forces(small_model, sp, xyz * s, np.asarray(box) * s)["E"][0]
        s[a] -= 2 * h
        em = orc.energy_forces(small_model, sp, xyz * s, np.asarray(box) * s)["E"][0]
        assert abs((ep - em) / (2 * h) - V[a, a]) < 2e-7 * r["virial_abs"]
    assert np.abs(V - V.T).max() < 1e-12 * r["virial_abs"]          # rotation invariance => symmetric
    assert np.allclose(r["F"], orc.energy_forces(small_model, sp, xyz, box)["F"], rtol=0, atol=1e-14)
    assert r["virial_abs"] >= np.abs(V).max()


def test_virial_full_tensor_and_clausius_form_nonperiodic(small_model):
    """Without a box every component follows from x -> (1 + eps) x, shear included, and V_ab = -sum_i x_ia F_ib."""
    sp, xyz, offs = inputs.molecule_batch(1, nmin=24, nmax=24, seed=31)
    r = orc.energy_forces_virial(small_model, sp, xyz, None)
    V, h = r["virial"], 2e-5
    for a in range(3):
        for b in range(3):
            eps = np.zeros((3, 3))
            eps[a, b] = h
            ep = orc.energy_forces(small_model, sp, xyz @ (np.eye(3) + eps), None)["E"][0]   # x'_b = x_b + eps_ab x_a
            em = orc.energy_forces(small_model, sp, xyz @ (np.eye(3) - eps), None)["E"][0]
            assert abs((ep - em) / (2 * h) - V[a, b]) < 2e-7 * r["virial_abs"], (a, b)
    assert np.abs(V + xyz.T @ r["F"]).max() < 1e-11 * r["virial_abs"]
    # a rigid translation changes nothing (net force is zero)
    r2 = orc.energy_forces_virial(small_model, sp, xyz + np.array([3.0, -2.0, 5.0]), None)
    assert np.abs(r2["virial"] - V).max() < 1e-10 * r["virial_abs"]


def test_virial_of_a_dimer_by_hand(small_model, consts):
    """Two atoms on the x axis: only V_xx = r dE/dr is non-zero, and dE/dr follows from the forces."""
    rr = 1.3
    sp = np.array([0, 3], dtype=np.int32)
    xyz = np.array([[0.0, 0.0, 0.0], [rr, 0.0, 0.0]])
    r = orc.energy_forces_virial(small_model, sp, xyz, None)
    dEdr = -r["F"][1, 0]
    assert abs(r["virial"][0, 0] - rr * dEdr) < 1e-12 * max(1.0, abs(rr * dEdr))
    V = r["virial"].copy()
    V[0, 0] = 0.0
    assert np.abs(V).max() < 1e-14


# ---------------------------------------------------------------- NEXT-2, second part: general (triclinic) cells, all periodic images
# SURVEY.md 8(f) item 2; PAPER.md L41 ("optionally cell vectors"), L49 (shift vectors), L307 (minimum image or all images).
def _small_water(n_waters, L, seed):
    return inputs.water_box(n_waters, L, seed=seed)


def test_cell_path_equals_box_path_for_a_wide_orthorhombic_cell(small_model, water64):
    """With every edge >= 2 R the all-images list IS the minimum-image list: the general-cell code must give the box code's
    numbers (catches a wrong shift sign, a transposed cell, a self-pair left in)."""
    sp, xyz, box = water64
    a = orc.energy_forces(small_model, sp, xyz, box, want_e_atom=True, want_aev=True)
    b = orc.energy_forces_cell(small_model, sp, xyz, np.diag(box), want_e_atom=True, want_aev=True, want_virial=True)
    assert abs(a["E"][0] - b["E"][0]) < 1e-10 * abs(a["E"][0])
    assert np.abs(a["F"] - b["F"]).max() < 1e-10 and np.abs(a["aev"] - b["aev"]).max() < 1e-12
    v = orc.energy_forces_virial(small_model, sp, xyz, box)
    assert np.abs(v["virial"] - b["virial"]).max() < 1e-11 * v["virial_abs"]
    # lists: every (j, 0-or-lattice shift) of the cell path is the box path's j, once
    lc = orc.neighbors_cell(xyz, np.diag(box), 5.1)
    lb = orc.neighbors(xyz, box, 5.1)
    for i in range(len(sp)):
        assert sorted(j for j, *_ in lc[i]) == sorted(lb[i])


def test_lattice_equivalent_cells_give_the_same_answer(small_model):
    """A lattice does not know which basis describes it: (a, b, c) -> (a, b + a, c + 2a - b) is unimodular, the cell becomes
    strongly triclinic, every energy and force must stay (catches any place where the code assumes an orthogonal cell or
    mixes up rows and columns of the cell matrix), for a wide cell and for one smaller than the cutoff."""
    for n_w, L, seed in ((27, 9.31, 3), (4, 4.9, 4)):
        sp, xyz, box = _small_water(n_w, L, seed)
        h = np.diag(box).astype(float)
        h2 = np.array([h[0], h[1] + h[0], h[2] + 2 * h[0] - h[1]])
        a = orc.energy_forces_cell(small_model, sp, xyz, h, want_virial=True)
        b = orc.energy_forces_cell(small_model, sp, xyz, h2, want_virial=True)
        assert abs(a["E"][0] - b["E"][0]) < 1e-10 * abs(a["E"][0])
        assert np.abs(a["F"] - b["F"]).max() < 1e-9
        assert np.abs(a["virial"] - b["virial"]).max() < 1e-10 * a["virial_abs"]
        # and the lists hold the same number of images per atom
        la, lb = orc.neighbors_cell(xyz, h, 5.1), orc.neighbors_cell(xyz, h2, 5.1)
        assert [len(r) for r in la] == [len(r) for r in lb]


def test_small_cell_all_images_equals_its_supercell_by_minimum_image(small_model):
    """All-images PBC in a cell below 2 R must equal the same crystal described by a supercell wide enough for the
    minimum image, evaluated by the ORTHORHOMBIC BOX code (a different code path): E_super = copies x E_cell and every
    image atom carries the force of its original.  L = 4.9 < R: atoms also see their own images."""
    for n_w, L, m, seed in ((27, 9.31, 2, 3), (4, 4.9, 3, 4)):
        sp, xyz, box = _small_water(n_w, L, seed)
        cell = orc.energy_forces_cell(small_model, sp, xyz, np.diag(box))
        shifts = np.array([[i, j, k] for i in range(m) for j in range(m) for k in range(m)], dtype=float) * np.asarray(box, dtype=float)
        xs = np.concatenate([xyz + s for s in shifts])
        sps = np.tile(sp, m ** 3)
        sup = orc.energy_forces(small_model, sps, xs, np.asarray(box) * m)
        assert abs(sup["E"][0] - m ** 3 * cell["E"][0]) < 1e-9 * abs(sup["E"][0])
        n = len(sp)
        for c in range(m ** 3):
            assert np.abs(sup["F"][c * n:(c + 1) * n] - cell["F"]).max() < 1e-9
    # the small cell really is in the regime the test is about: more images than atoms, self images included
    lst = orc.neighbors_cell(xyz, np.diag(box), 5.1)
    assert any(j == i for i, row in enumerate(lst) for j, *_ in row) and min(len(r) for r in lst) > len(sp)


def test_all_images_list_against_explicit_images_and_kdtree():
    """Lists of a skewed small cell against scipy's KD-tree over explicitly generated images (an independent search)."""
    rng = np.random.default_rng(8)
    h = np.array([[6.0, 0.0, 0.0], [2.2, 5.5, 0.0], [-1.3, 1.9, 6.4]])
    xyz = rng.random((40, 3)) @ h + rng.integers(-2, 3, size=(40, 3)) @ h     # unwrapped coordinates
    lst = orc.neighbors_cell(xyz, h, 5.1)
    S = np.array([[i, j, k] for i in range(-7, 8) for j in range(-7, 8) for k in range(-7, 8)])
    img = (xyz[None, :, :] + (S @ h)[:, None, :]).reshape(-1, 3)
    tree = cKDTree(img)
    for i in range(40):
        near = tree.query_ball_point(xyz[i], 5.1 - 1e-12)
        ref = sorted((q % 40, *S[q // 40]) for q in near if not (q % 40 == i and not S[q // 40].any()))
        assert [tuple(int(v) for v in r) for r in ref] == lst[i]


def test_triclinic_forces_and_sheared_virial_by_finite_differences(small_model):
    """A genuinely triclinic small cell (a sheared, squeezed water cell - not a re-description of a cubic one): forces are
    minus the energy gradient, and the FULL virial tensor, shear components included, is the derivative of the energy under
    the homogeneous deformation x -> x (1 + eps), cell -> cell (1 + eps) (the first part of the row pinned
    only the diagonal under PBC)."""
    sp, xyz, box = _small_water(8, 6.2, 6)
    D = np.array([[1.0, 0.0, 0.0], [0.23, 0.94, 0.0], [-0.17, 0.12, 1.05]])
    x = xyz @ D
    h = np.diag(box) @ D
    r = orc.energy_forces_cell(small_model, sp, x, h, want_virial=True)
    rng = np.random.default_rng(0)
    for i in rng.choice(len(sp), 6, replace=False):
        for c in range(3):
            xp, xm = x.copy(), x.copy()
            xp[i, c] += 1e-4
            xm[i, c] -= 1e-4
            g = (orc.energy_forces_cell(small_model, sp, xp, h, want_forces=False)["E"][0]
                 - orc.energy_forces_cell(small_model, sp, xm, h, want_forces=False)["E"][0]) / 2e-4
            assert abs(-g - r["F"][i, c]) < 2e-6 * max(1.0, np.abs(r["F"]).max())
    e = 2e-5
    for a in range(3):
        for b in range(3):
            eps = np.zeros((3, 3))
            eps[a, b] = e
            Ep = orc.energy_forces_cell(small_model, sp, x @ (np.eye(3) + eps), h @ (np.eye(3) + eps), want_forces=False)["E"][0]
            Em = orc.energy_forces_cell(small_model, sp, x @ (np.eye(3) - eps), h @ (np.eye(3) - eps), want_forces=False)["E"][0]
            assert abs((Ep - Em) / (2 * e) - r["virial"][a, b]) < 3e-7 * r["virial_abs"], (a, b)
    assert np.abs(r["virial"] - r["virial"].T).max() < 1e-11 * r["virial_abs"]
    assert np.abs(r["F"].sum(0)).max() < 1e-9


def test_cell_rotation_covariance_and_md_reduces_to_box_md(small_model):
    """Rotating cell and coordinates together leaves E and rotates F; orc_md_cell on a wide diagonal cell is orc_md."""
    sp, xyz, box = _small_water(8, 6.2, 6)
    h = np.diag(box) @ np.array([[1.0, 0.0, 0.0], [0.2, 1.0, 0.0], [0.1, -0.15, 1.0]])
    R = rot(4)
    a = orc.energy_forces_cell(small_model, sp, xyz, h)
    b = orc.energy_forces_cell(small_model, sp, xyz @ R.T, h @ R.T)
    assert abs(a["E"][0] - b["E"][0]) < 1e-10 * abs(a["E"][0]) and np.abs(a["F"] @ R.T - b["F"]).max() < 1e-9
    sp, xyz, box = inputs.water_box(64, 12.42, seed=inputs.SEED0 + 1)
    v = inputs.maxwell_boltzmann(sp, 300.0, seed=3)
    m1 = orc.md(small_model, sp, xyz, v, inputs.MASS, box, 0.5, inputs.ACCEL_CONV, 3)
    m2 = orc.md_cell(small_model, sp, xyz, v, inputs.MASS, np.diag(box), 0.5, inputs.ACCEL_CONV, 3)
    assert np.abs(m1["xyz"] - m2["xyz"]).max() < 1e-12 and np.abs(m1["epot"] - m2["epot"]).max() < 1e-9
