"""Seeded synthetic inputs shared by the oracle-side tests and the CUDA-side tests / bench.

This module holds NONE of the method's arithmetic (no cutoff function, no AEV term, no MLP, no
integrator): only model constants, random weights and geometry generators.  Both the oracle and the
CUDA path receive what is generated here as plain arrays.

Constants: PAPER.md prints none of the ANI-2x hyper-parameters (SURVEY.md 8(c) reading A2); the values
below are the published ANI-2x ones as recalled there and are create-time parameters on both sides.
Workloads: stand-ins for the paper's water boxes (648 -> 500K atoms) and solvated DHFR (~20K atoms),
PAPER.md L323; recipes in DESIGN.md "Input recipe" / BASELINE.json configs 1-5.
"""
import math

import numpy as np
from scipy.spatial import cKDTree

SPECIES = ("H", "C", "N", "O", "S", "F", "Cl")           # reading B2: index order 0..6
MASS = np.array([1.008, 12.011, 14.007, 15.999, 32.06, 18.998, 35.45])   # amu (reading B6)
ACCEL_CONV = 4.184e-4            # (kcal/mol/A)/amu -> A/fs^2
KB = 0.0019872041                # kcal/mol/K
WATER_DENSITY = 0.033428         # molecules / A^3 (1 g/cm^3)
SEED0 = 240501491
# Reading B7: scalar applied to the last-layer weights so that random Xavier weights give liquid-like force
# magnitudes on water.  Derived with the oracle only (tests/golden/force_scale.md): RMS |F| = 0.30 at scale 1.
FORCE_SCALE_WATER = 66.0
# MD workloads (bench.py): random weights are not a bound liquid, and at scale 66 the box heats from 300 K to
# > 4000 K within 200 steps (measured on the B200).  At scale 2 the kinetic
# temperature stays at 300-320 K over 1000 steps and the list is rebuilt every ~6.7 steps, the cadence of
# thermal water with a 0.5 A skin (SURVEY.md 8(c) C2 expects 6-12).
FORCE_SCALE_MD = 2.0

# BASELINE.json layer widths, species order H C N O S F Cl
WIDTHS = np.array([
    [1008, 256, 192, 160, 1],
    [1008, 224, 192, 160, 1],
    [1008, 192, 160, 128, 1],
    [1008, 192, 160, 128, 1],
    [1008, 160, 128, 96, 1],
    [1008, 160, 128, 96, 1],
    [1008, 160, 128, 96, 1],
], dtype=np.int32)


def ani2x_constants():
    """Reading A1/A2: cutoffs 5.1 / 3.5 A; 16 radial shifts, 8 angular radial shifts, 4 angle shifts."""
    return dict(
        rcr=5.1, rca=3.5,
        eta_r=19.7, shf_r=0.8 + 0.26875 * np.arange(16),
        eta_a=12.5, zeta=14.1, shf_a=0.8 + 0.3375 * np.arange(8),
        shf_z=(2 * np.arange(4) + 1) * math.pi / 8,
        celu_alpha=0.1,
    )


def make_weights(seed, n_nets=1, widths=WIDTHS, last_layer_scale=1.0, bias_std=0.0):
    """Reading B3: Xavier-normal W ~ N(0, 2/(fan_in+fan_out)), b = 0 (bias_std > 0 only for tests).

    Flat fp32-representable fp64 array, order [net][species][layer](W[in][out] row-major, b[out]).
    Values are rounded to fp32 so that both sides load bit-identical numbers.
    """
    rng = np.random.default_rng(seed)
    out = []
    nl = widths.shape[1] - 1
    for _ in range(n_nets):
        for s in range(widths.shape[0]):
            for l in range(nl):
                fi, fo = int(widths[s, l]), int(widths[s, l + 1])
                W = rng.normal(0.0, math.sqrt(2.0 / (fi + fo)), size=(fi, fo))
                b = rng.normal(0.0, bias_std, size=fo) if bias_std > 0 else np.zeros(fo)
                if l == nl - 1:
                    W = W * last_layer_scale
                out.append(W.ravel())
                out.append(b)
    return np.concatenate(out).astype(np.float32).astype(np.float64)


# ------------------------------------------------------------------------------------------------
# geometry
# ------------------------------------------------------------------------------------------------
def _random_rotations(rng, n):
    q = rng.normal(size=(n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    w, x, y, z = q.T
    R = np.empty((n, 3, 3))
    R[:, 0, 0] = 1 - 2 * (y * y + z * z); R[:, 0, 1] = 2 * (x * y - z * w); R[:, 0, 2] = 2 * (x * z + y * w)
    R[:, 1, 0] = 2 * (x * y + z * w); R[:, 1, 1] = 1 - 2 * (x * x + z * z); R[:, 1, 2] = 2 * (y * z - x * w)
    R[:, 2, 0] = 2 * (x * z - y * w); R[:, 2, 1] = 2 * (y * z + x * w); R[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return R


def _rsa_points(rng, n_target, L, dmin, forbidden=None, forbidden_r=0.0, max_rounds=100000):
    """Random sequential addition of points in a periodic cube with minimum-image separation >= dmin.

    Batched: candidates are drawn uniformly, those closer than dmin to an accepted point (or than
    forbidden_r to a forbidden point) are rejected, the rest are accepted greedily in draw order.
    """
    pts = np.empty((0, 3))
    ftree = cKDTree(np.mod(forbidden, L), boxsize=L) if forbidden is not None and len(forbidden) else None
    for _ in range(max_rounds):
        need = n_target - len(pts)
        if need <= 0:
            break
        cand = rng.uniform(0.0, L, size=(max(64, 2 * need), 3))
        if ftree is not None:
            d, _ = ftree.query(cand, k=1)
            cand = cand[d >= forbidden_r]
        if len(pts):
            d, _ = cKDTree(pts, boxsize=L).query(cand, k=1)
            cand = cand[d >= dmin]
        if len(cand) == 0:
            continue
        pairs = cKDTree(cand, boxsize=L).query_pairs(dmin, output_type="ndarray")
        keep = np.ones(len(cand), dtype=bool)
        if len(pairs):
            order = np.lexsort((pairs[:, 0], pairs[:, 1]))
            for a, b in pairs[order]:          # a < b: drop the later draw if the earlier survives
                if keep[a]:
                    keep[b] = False
        pts = np.vstack([pts, cand[keep][:need]])
    if len(pts) < n_target:
        raise RuntimeError("RSA did not converge")
    return pts


def _waters_from_oxygens(rng, O):
    """Rigid water: O-H 0.9572 A, H-O-H 104.52 deg, uniform random orientation.  Order per molecule: O,H,H."""
    n = len(O)
    half = math.radians(104.52) / 2
    h1 = 0.9572 * np.array([math.sin(half), 0.0, math.cos(half)])
    h2 = 0.9572 * np.array([-math.sin(half), 0.0, math.cos(half)])
    R = _random_rotations(rng, n)
    xyz = np.empty((n, 3, 3))
    xyz[:, 0] = O
    xyz[:, 1] = O + R @ h1
    xyz[:, 2] = O + R @ h2
    species = np.tile(np.array([3, 0, 0], dtype=np.int32), n)
    return species, xyz.reshape(-1, 3)


def water_box(n_waters, L=None, seed=SEED0, dmin=2.5):
    """Configs 1-3: n rigid waters in a periodic cube at 1 g/cm^3 (L = (n/rho)^(1/3) unless given).

    Returns species int32[3n], xyz float64[3n,3] (fp32-representable), box float64[3].
    """
    if L is None:
        L = (n_waters / WATER_DENSITY) ** (1.0 / 3.0)
    rng = np.random.default_rng(seed)
    O = _rsa_points(rng, n_waters, L, dmin)
    species, xyz = _waters_from_oxygens(rng, O)
    xyz = xyz.astype(np.float32).astype(np.float64)
    L = float(np.float32(L))
    return species, xyz, np.array([L, L, L])


def maxwell_boltzmann(species, T=300.0, seed=SEED0 + 100):
    """Reading C3: sigma = sqrt(kB T / m) per component (A/fs), centre-of-mass velocity removed."""
    rng = np.random.default_rng(seed)
    m = MASS[species]
    v = rng.normal(size=(len(species), 3)) * np.sqrt(KB * T * ACCEL_CONV / m)[:, None]
    v -= (m[:, None] * v).sum(0) / m.sum()
    return v.astype(np.float32).astype(np.float64)


def _chain(rng, n_atoms, L, dmin, bond=(1.0, 1.5), max_tries=2000, block=64):
    """Self-avoiding periodic random-walk chain: bond length U(bond), uniform direction, every atom
    except the bonded predecessor at minimum-image distance >= dmin."""
    pts = np.zeros((n_atoms, 3))
    pts[0] = rng.uniform(0, L, 3)
    tree, tree_n = None, 0

    def ok(p, i):
        if tree is not None:
            for idx in tree.query_ball_point(np.mod(p, L), dmin):
                if idx != i - 1:
                    return False
        d = pts[tree_n:i] - p
        d -= L * np.round(d / L)
        r2 = np.einsum("ij,ij->i", d, d)
        if i - 1 >= tree_n:
            r2[i - 1 - tree_n] = np.inf
        return bool((r2 >= dmin * dmin).all())

    i = 1
    while i < n_atoms:
        placed = False
        for _ in range(max_tries):
            d = rng.normal(size=3)
            d /= np.linalg.norm(d)
            p = pts[i - 1] + d * rng.uniform(*bond)
            if ok(p, i):
                pts[i] = p
                placed = True
                break
        if placed:
            i += 1
            if i - tree_n >= block:
                tree, tree_n = cKDTree(np.mod(pts[:i], L), boxsize=L), i
        else:                                   # dead end: back up 5 atoms
            i = max(1, i - 5)
            if i < tree_n:
                tree_n = i
                tree = cKDTree(np.mod(pts[:i], L), boxsize=L) if i > 0 else None
    t = cKDTree(np.mod(pts, L), boxsize=L)
    pairs = t.query_pairs(dmin * 0.999999, output_type="ndarray")
    if any(abs(int(a) - int(b)) != 1 for a, b in pairs):
        raise RuntimeError("chain self-avoidance violated")
    return pts


def solvated_chain(n_solute=4000, L=62.0, seed=SEED0 + 4):
    """Config 4: random-walk solute (H .50 C .31 N .08 O .09 S .01 F .005 Cl .005; bonds 1.0-1.5 A;
    non-bonded >= 2.2 A) in rigid water at 1 g/cm^3; waters whose O is within 2.2 A of a solute atom removed
    (about 21,100 atoms)."""
    rng = np.random.default_rng(seed)
    solute = _chain(rng, n_solute, L, 2.2)
    sp_sol = rng.choice(7, size=n_solute, p=[0.50, 0.31, 0.08, 0.09, 0.01, 0.005, 0.005]).astype(np.int32)
    n_w = int(round(WATER_DENSITY * L ** 3))
    O = _rsa_points(rng, n_w, L, 2.5)
    d, _ = cKDTree(np.mod(solute, L), boxsize=L).query(O, k=1)
    O = O[d >= 2.2]
    sp_w, xyz_w = _waters_from_oxygens(rng, O)
    species = np.concatenate([sp_sol, sp_w])
    xyz = np.vstack([solute, xyz_w]).astype(np.float32).astype(np.float64)
    L = float(np.float32(L))
    return species, xyz, np.array([L, L, L])


def molecule_batch(n_mols=8192, nmin=8, nmax=30, seed=SEED0 + 5):
    """Config 5: non-periodic chain molecules, n ~ U{nmin..nmax}, species iid
    H .5 C .3 N .07 O .08 F .02 S .02 Cl .01, bonds U(1.0,1.5) A, all atoms >= 1.1 A apart.
    Returns species, xyz, mol_offsets int32[n_mols+1]."""
    rng = np.random.default_rng(seed)
    sizes = rng.integers(nmin, nmax + 1, size=n_mols)
    offs = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int32)
    # species index order H C N O S F Cl -> probabilities for (H,C,N,O,S,F,Cl)
    p = [0.5, 0.3, 0.07, 0.08, 0.02, 0.02, 0.01]
    species = rng.choice(7, size=offs[-1], p=p).astype(np.int32)
    xyz = np.zeros((offs[-1], 3))
    for m in range(n_mols):
        n = sizes[m]
        pts = np.zeros((n, 3))
        i = 1
        while i < n:
            ok = False
            for _ in range(200):
                d = rng.normal(size=3)
                d /= np.linalg.norm(d)
                q = pts[i - 1] + d * rng.uniform(1.0, 1.5)
                dd = pts[:i - 1] - q if i > 1 else np.zeros((0, 3))
                if len(dd) == 0 or (np.einsum("ij,ij->i", dd, dd) >= 1.1 * 1.1).all():
                    pts[i] = q
                    ok = True
                    break
            i = i + 1 if ok else max(1, i - 3)
        xyz[offs[m]:offs[m + 1]] = pts + rng.uniform(-20, 20, 3)
    return species, xyz.astype(np.float32).astype(np.float64), offs


def dense_box(density, L=12.0, dmin=1.2, seed=SEED0 + 6, n_species=7):
    """Compressed mixed-species periodic box (not a workload of the paper: a stress case for the neighbour capacities):
    `density` atoms / A^3 by random sequential addition with separation >= dmin, species iid uniform.
    density 0.25 => ~45 neighbours inside 3.5 A and ~139 inside 5.1 A per atom (water: 18 / 56)."""
    rng = np.random.default_rng(seed)
    n = int(round(density * L ** 3))
    xyz = _rsa_points(rng, n, L, dmin).astype(np.float32).astype(np.float64)
    species = rng.integers(0, n_species, size=n).astype(np.int32)
    species[:n_species] = np.arange(n_species)
    L = float(np.float32(L))
    return species, xyz, np.array([L, L, L])


def replicate(species, xyz, box, k):
    """k x k x k periodic images of a box (extensivity pin)."""
    sh = np.array([[a, b, c] for a in range(k) for b in range(k) for c in range(k)], dtype=np.float64) * box
    xyz_r = (xyz[None, :, :] + sh[:, None, :]).reshape(-1, 3)
    return np.tile(species, k ** 3), xyz_r, box * k
