"""ctypes loader for oracle/nnp_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import
this module.  It imports nothing from paper_2405_01491_b200 (the CUDA path) and the CUDA path imports
nothing from here.  All arithmetic of the method lives in nnp_oracle.c; this file only marshals numpy
arrays (fp64) into the C calls.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "nnp_oracle.c")
_LIB = os.path.join(_HERE, "libnnp_oracle.so")
_lib = None


def build(force=False):
    """gcc -O2, fp64, no FMA contraction (the fp32 list predicate of reading A3 needs separate ops)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
               _SRC, "-o", _LIB, "-lm"]
        subprocess.check_call(cmd)
    return _LIB


class _Model(C.Structure):
    _fields_ = [
        ("n_species", C.c_int), ("rcr", C.c_double), ("rca", C.c_double),
        ("eta_r", C.c_double), ("n_shf_r", C.c_int), ("shf_r", C.POINTER(C.c_double)),
        ("eta_a", C.c_double), ("zeta", C.c_double), ("n_shf_a", C.c_int), ("shf_a", C.POINTER(C.c_double)),
        ("n_shf_z", C.c_int), ("shf_z", C.POINTER(C.c_double)),
        ("celu_alpha", C.c_double), ("n_nets", C.c_int), ("n_layers", C.c_int),
        ("widths", C.POINTER(C.c_int)), ("params", C.POINTER(C.c_double)),
        ("self_energy", C.POINTER(C.c_double)),
    ]


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double)) if a is not None else None


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int)) if a is not None else None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.orc_aev_len.restype = C.c_int
        L.orc_pair_index.restype = C.c_int
        L.orc_params_per_net.restype = C.c_long
        L.orc_fc.restype = C.c_double
        L.orc_fc.argtypes = [C.c_double, C.c_double]
        L.orc_celu.restype = C.c_double
        L.orc_celu.argtypes = [C.c_double, C.c_double]
        L.orc_mlp.restype = C.c_double
        L.orc_neighbors_brute.argtypes = [C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_int),
                                          C.c_double, C.c_int, C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_int)]
        L.orc_neighbors_grid.argtypes = [C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double),
                                         C.c_double, C.c_int, C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_int)]
        L.orc_needs_rebuild.argtypes = [C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_double]
        L.orc_md.argtypes = [C.POINTER(_Model), C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_double),
                             C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_int, C.POINTER(C.c_double),
                             C.POINTER(C.c_double), C.c_double, C.c_double, C.c_int, C.c_double, C.c_int,
                             C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_int)]
        L.orc_md_cell.argtypes = [C.POINTER(_Model), C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_double),
                                  C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_int, C.POINTER(C.c_double),
                                  C.POINTER(C.c_double), C.c_double, C.c_double, C.c_int, C.c_double,
                                  C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_int)]
        L.orc_neighbors_cell.argtypes = [C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_int),
                                         C.c_double, C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_int)]
        L.orc_energy_forces_cell.argtypes = [C.POINTER(_Model), C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_double),
                                             C.POINTER(C.c_double), C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_double),
                                             C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_double),
                                             C.POINTER(C.c_double)]
        _lib = L
    return _lib


class OracleModel:
    """Holds the model constants and flat weights as fp64 arrays for the C oracle.

    consts: dict with rcr, rca, eta_r, shf_r, eta_a, zeta, shf_a, shf_z, celu_alpha.
    widths: int array [S][n_layers+1].  params: flat array, [net][species][layer](W[in][out], b[out]).
    """

    def __init__(self, consts, widths, params, n_nets=1, self_energy=None):
        self.widths = np.ascontiguousarray(widths, dtype=np.int32)
        self.S, nl1 = self.widths.shape
        self.shf_r = np.ascontiguousarray(consts["shf_r"], dtype=np.float64)
        self.shf_a = np.ascontiguousarray(consts["shf_a"], dtype=np.float64)
        self.shf_z = np.ascontiguousarray(consts["shf_z"], dtype=np.float64)
        self.params = np.ascontiguousarray(params, dtype=np.float64)
        self.self_energy = None if self_energy is None else np.ascontiguousarray(self_energy, dtype=np.float64)
        m = _Model()
        m.n_species = self.S
        m.rcr, m.rca = float(consts["rcr"]), float(consts["rca"])
        m.eta_r, m.n_shf_r, m.shf_r = float(consts["eta_r"]), len(self.shf_r), _dp(self.shf_r)
        m.eta_a, m.zeta = float(consts["eta_a"]), float(consts["zeta"])
        m.n_shf_a, m.shf_a = len(self.shf_a), _dp(self.shf_a)
        m.n_shf_z, m.shf_z = len(self.shf_z), _dp(self.shf_z)
        m.celu_alpha = float(consts["celu_alpha"])
        m.n_nets, m.n_layers = int(n_nets), nl1 - 1
        m.widths, m.params = _ip(self.widths), _dp(self.params)
        m.self_energy = _dp(self.self_energy)
        self.c = m
        self.n_nets = int(n_nets)
        self.aev_len = lib().orc_aev_len(C.byref(m))
        per_net = lib().orc_params_per_net(C.byref(m))
        assert self.params.size == per_net * self.n_nets, (self.params.size, per_net, n_nets)

    def mlp(self, net, species, G, want_grad=False):
        G = np.ascontiguousarray(G, dtype=np.float64)
        grad = np.zeros_like(G) if want_grad else None
        e = lib().orc_mlp(C.byref(self.c), C.c_int(net), C.c_int(species), _dp(G), _dp(grad))
        return (e, grad) if want_grad else e


def pair_index(S, s, t):
    return lib().orc_pair_index(C.c_int(S), C.c_int(s), C.c_int(t))


def fc(r, R):
    return lib().orc_fc(r, R)


def celu(x, alpha):
    return lib().orc_celu(x, alpha)


def num_threads():
    return lib().orc_num_threads()


def neighbors(xyz, box, rcut, mol_id=None, fp32_pred=False, method="brute", cap=256):
    """Directed neighbour rows as a list of sorted int arrays (O1)."""
    xyz = np.ascontiguousarray(xyz, dtype=np.float64)
    n = xyz.shape[0]
    boxa = None if box is None else np.ascontiguousarray(box, dtype=np.float64)
    mid = None if mol_id is None else np.ascontiguousarray(mol_id, dtype=np.int32)
    while True:
        counts = np.zeros(max(n, 1), dtype=np.int32)
        lst = np.zeros((max(n, 1), cap), dtype=np.int32)
        if method == "grid":
            rc = lib().orc_neighbors_grid(n, _dp(xyz), _dp(boxa), float(rcut), int(fp32_pred), cap, _ip(counts), _ip(lst))
        else:
            rc = lib().orc_neighbors_brute(n, _dp(xyz), _dp(boxa), _ip(mid), float(rcut), int(fp32_pred), cap,
                                           _ip(counts), _ip(lst))
        if rc <= -1000000000:
            raise ValueError("box smaller than 2*rcut")
        if rc >= 0:
            break
        cap = -rc + 8
    return [np.sort(lst[i, :counts[i]]) for i in range(n)]


def energy_forces(model, species, xyz, box=None, mol_offsets=None, nbr_method=0,
                  want_forces=True, want_e_atom=False, want_aev=False, want_dEdG=False):
    """O1-O6.  Returns dict(E[n_mols], F[n,3], e_atom[n], aev[n,len], dEdG[n,len])."""
    species = np.ascontiguousarray(species, dtype=np.int32)
    xyz = np.ascontiguousarray(xyz, dtype=np.float64)
    n = xyz.shape[0]
    boxa = None if box is None else np.ascontiguousarray(box, dtype=np.float64)
    mo = None if mol_offsets is None else np.ascontiguousarray(mol_offsets, dtype=np.int32)
    n_mols = 1 if mo is None else len(mo) - 1
    E = np.zeros(n_mols)
    F = np.zeros((n, 3)) if want_forces else None
    ea = np.zeros(n) if want_e_atom else None
    aev = np.zeros((n, model.aev_len)) if want_aev else None
    dg = np.zeros((n, model.aev_len)) if want_dEdG else None
    rc = lib().orc_energy_forces(C.byref(model.c), C.c_int(n), _ip(species), _dp(xyz), _dp(boxa), C.c_int(n_mols),
                                 _ip(mo), C.c_int(nbr_method), _dp(E), _dp(F), _dp(ea), _dp(aev), _dp(dg))
    if rc != 0:
        raise RuntimeError("orc_energy_forces failed: %d" % rc)
    return {"E": E, "F": F, "e_atom": ea, "aev": aev, "dEdG": dg}


def energy_forces_cell(model, species, xyz, cell, mol_offsets=None, want_forces=True, want_e_atom=False, want_aev=False,
                       want_virial=False):
    """O1-O6 in a general cell (rows of cell[3][3] = lattice vectors) with ALL periodic images.
    Returns dict(E[n_mols], F[n,3], e_atom[n], aev[n,len], virial[3,3], virial_abs)."""
    species = np.ascontiguousarray(species, dtype=np.int32)
    xyz = np.ascontiguousarray(xyz, dtype=np.float64)
    n = xyz.shape[0]
    cella = np.ascontiguousarray(cell, dtype=np.float64).reshape(9)
    mo = None if mol_offsets is None else np.ascontiguousarray(mol_offsets, dtype=np.int32)
    n_mols = 1 if mo is None else len(mo) - 1
    E = np.zeros(n_mols)
    F = np.zeros((n, 3)) if (want_forces or want_virial) else None
    ea = np.zeros(n) if want_e_atom else None
    aev = np.zeros((n, model.aev_len)) if want_aev else None
    vir = np.zeros(10) if want_virial else None
    rc = lib().orc_energy_forces_cell(C.byref(model.c), C.c_int(n), _ip(species), _dp(xyz), _dp(cella), C.c_int(n_mols),
                                      _ip(mo), _dp(E), _dp(F), _dp(ea), _dp(aev), _dp(vir))
    if rc != 0:
        raise RuntimeError("orc_energy_forces_cell failed: %d" % rc)
    out = {"E": E, "F": F, "e_atom": ea, "aev": aev}
    if want_virial:
        out["virial"], out["virial_abs"] = vir[:9].reshape(3, 3).copy(), float(vir[9])
    return out


def neighbors_cell(xyz, cell, rcut, mol_id=None):
    """All-images lists in a general cell: per atom a sorted list of (j, s0, s1, s2)."""
    xyz = np.ascontiguousarray(xyz, dtype=np.float64)
    n = xyz.shape[0]
    cella = np.ascontiguousarray(cell, dtype=np.float64).reshape(9)
    mid = None if mol_id is None else np.ascontiguousarray(mol_id, dtype=np.int32)
    cap = 128
    while True:
        counts = np.zeros(n, dtype=np.int32)
        lst = np.zeros((n, cap), dtype=np.int32)
        shf = np.zeros((n, cap, 3), dtype=np.int32)
        rc = lib().orc_neighbors_cell(n, _dp(xyz), _dp(cella), _ip(mid), float(rcut), cap, _ip(counts), _ip(lst), _ip(shf))
        if rc >= 0:
            break
        if rc <= -1000000000:
            raise RuntimeError("singular cell")
        cap = -rc + 8
    return [sorted((int(lst[i, k]), int(shf[i, k, 0]), int(shf[i, k, 1]), int(shf[i, k, 2])) for k in range(counts[i])) for i in range(n)]


def md_cell(model, species, xyz, vel, mass, cell, dt, accel_conv, n_steps, skin=0.5):
    """O7 velocity Verlet in a general cell with all images."""
    species = np.ascontiguousarray(species, dtype=np.int32)
    x = np.array(xyz, dtype=np.float64, order="C")
    v = np.array(vel, dtype=np.float64, order="C")
    n = x.shape[0]
    F = np.zeros((n, 3))
    mass = np.ascontiguousarray(mass, dtype=np.float64)
    cella = np.ascontiguousarray(cell, dtype=np.float64).reshape(9)
    epot = np.zeros(n_steps + 1)
    ekin = np.zeros(n_steps + 1)
    nreb = C.c_int(0)
    rc = lib().orc_md_cell(C.byref(model.c), n, _ip(species), _dp(x), _dp(v), _dp(F), 0, _dp(mass), _dp(cella), float(dt),
                           float(accel_conv), int(n_steps), float(skin), _dp(epot), _dp(ekin), C.byref(nreb))
    if rc != 0:
        raise RuntimeError("orc_md_cell failed: %d" % rc)
    return {"xyz": x, "vel": v, "F": F, "epot": epot, "ekin": ekin, "n_rebuilds": nreb.value}


def needs_rebuild(xyz, xref, skin):
    xyz = np.ascontiguousarray(xyz, dtype=np.float64)
    xref = np.ascontiguousarray(xref, dtype=np.float64)
    return bool(lib().orc_needs_rebuild(xyz.shape[0], _dp(xyz), _dp(xref), float(skin)))


def md(model, species, xyz, vel, mass, box, dt, accel_conv, n_steps, skin=0.5, nbr_method=0, forces=None):
    """O7 velocity Verlet.  Returns dict(xyz, vel, F, epot[n_steps+1], ekin[n_steps+1], n_rebuilds)."""
    species = np.ascontiguousarray(species, dtype=np.int32)
    x = np.array(xyz, dtype=np.float64, order="C")
    v = np.array(vel, dtype=np.float64, order="C")
    n = x.shape[0]
    F = np.zeros((n, 3)) if forces is None else np.array(forces, dtype=np.float64, order="C")
    mass = np.ascontiguousarray(mass, dtype=np.float64)
    boxa = None if box is None else np.ascontiguousarray(box, dtype=np.float64)
    epot = np.zeros(n_steps + 1)
    ekin = np.zeros(n_steps + 1)
    nreb = C.c_int(0)
    rc = lib().orc_md(C.byref(model.c), n, _ip(species), _dp(x), _dp(v), _dp(F), int(forces is not None), _dp(mass),
                      _dp(boxa), float(dt), float(accel_conv), int(n_steps), float(skin), int(nbr_method),
                      _dp(epot), _dp(ekin), C.byref(nreb))
    if rc != 0:
        raise RuntimeError("orc_md failed: %d" % rc)
    return {"xyz": x, "vel": v, "F": F, "epot": epot, "ekin": ekin, "n_rebuilds": nreb.value}


def philox4x32_10(ctr, key):
    """Philox4x32-10 block (4 x uint32) for counter ctr[4] and key[2]; test hook of the Langevin generator."""
    c = (C.c_uint32 * 4)(*[int(x) & 0xffffffff for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) & 0xffffffff for x in key])
    out = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, out)
    return [int(x) for x in out]


def langevin_normals(atom, step, seed):
    xi = (C.c_double * 3)()
    lib().orc_langevin_normals(C.c_uint32(atom), C.c_uint32(step), C.c_uint64(seed), xi)
    return np.array(list(xi))


def md_langevin(model, species, xyz, vel, mass, box, dt, accel_conv, n_steps, gamma, kT, seed, step0=0, skin=0.5,
                nbr_method=0, forces=None):
    """NEXT-1: BAOAB Langevin dynamics.  Returns the same dict as md()."""
    species = np.ascontiguousarray(species, dtype=np.int32)
    x = np.array(xyz, dtype=np.float64, order="C")
    v = np.array(vel, dtype=np.float64, order="C")
    n = x.shape[0]
    F = np.zeros((n, 3)) if forces is None else np.array(forces, dtype=np.float64, order="C")
    mass = np.ascontiguousarray(mass, dtype=np.float64)
    boxa = None if box is None else np.ascontiguousarray(box, dtype=np.float64)
    epot = np.zeros(n_steps + 1)
    ekin = np.zeros(n_steps + 1)
    nreb = C.c_int(0)
    f = lib().orc_md_langevin
    f.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p,
                  C.c_double, C.c_double, C.c_int, C.c_double, C.c_int, C.c_double, C.c_double, C.c_uint64, C.c_uint32,
                  C.c_void_p, C.c_void_p, C.c_void_p]
    rc = f(C.cast(C.byref(model.c), C.c_void_p), n, species.ctypes.data, x.ctypes.data, v.ctypes.data, F.ctypes.data,
           int(forces is not None), mass.ctypes.data, None if boxa is None else boxa.ctypes.data, float(dt),
           float(accel_conv), int(n_steps), float(skin), int(nbr_method), float(gamma), float(kT), int(seed), int(step0),
           epot.ctypes.data, ekin.ctypes.data, C.cast(C.byref(nreb), C.c_void_p))
    if rc != 0:
        raise RuntimeError("orc_md_langevin failed: %d" % rc)
    return {"xyz": x, "vel": v, "F": F, "epot": epot, "ekin": ekin, "n_rebuilds": nreb.value}


def energy_forces_virial(model, species, xyz, box, nbr_method=0):
    """NEXT-2: E, F and the virial V_ab = dE/d eps_ab = sum_d d_a (dE/dd)_b of ONE structure.
    Returns dict(E, F, virial[3][3], virial_abs)."""
    species = np.ascontiguousarray(species, dtype=np.int32)
    x = np.ascontiguousarray(xyz, dtype=np.float64)
    n = x.shape[0]
    boxa = None if box is None else np.ascontiguousarray(box, dtype=np.float64)
    E = np.zeros(1)
    F = np.zeros((n, 3))
    W = np.zeros(10)
    f = lib().orc_energy_forces_virial
    f.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
    rc = f(C.cast(C.byref(model.c), C.c_void_p), n, species.ctypes.data, x.ctypes.data,
           None if boxa is None else boxa.ctypes.data, int(nbr_method), E.ctypes.data, F.ctypes.data, W.ctypes.data)
    if rc != 0:
        raise RuntimeError("orc_energy_forces_virial failed: %d" % rc)
    return {"E": E, "F": F, "virial": W[:9].reshape(3, 3).copy(), "virial_abs": float(W[9])}
