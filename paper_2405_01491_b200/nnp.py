"""Thin ctypes binding over the C-ABI library (include/nnp.h): same names, argument marshalling only.

Device arguments are torch CUDA tensors (PyTorch supplies device memory and the stream; every step of the
path runs in the library's kernels); host arguments of the *_host entry points are numpy arrays or pinned
CPU tensors.  There is no CPU fallback: if the library is missing or cannot be loaded, importing a symbol
raises.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libnnp_b200.so")

NNP_OK, NNP_EINVAL, NNP_ENOMEM, NNP_ECUDA, NNP_ECAPACITY, NNP_ESTALE, NNP_EBOX, NNP_ERANGE = 0, -1, -2, -3, -4, -5, -6, -7
NNP_MM_FP32_SIMT, NNP_MM_3XTF32_TC, NNP_MM_TF32_TC, NNP_MM_FP64_SIMT, NNP_MM_3XF16_TC = 0, 1, 2, 3, 4
STATUS_NAMES = {0: "NNP_OK", -1: "NNP_EINVAL", -2: "NNP_ENOMEM", -3: "NNP_ECUDA", -4: "NNP_ECAPACITY",
                -5: "NNP_ESTALE", -6: "NNP_EBOX", -7: "NNP_ERANGE"}

EXPORTS = ["nnp_create", "nnp_destroy", "nnp_last_error", "nnp_set_system", "nnp_set_system_cell", "nnp_set_positions",
           "nnp_build_neighbors", "nnp_get_neighbors", "nnp_energy_forces", "nnp_get_aev",
           "nnp_get_atomic_energies", "nnp_md_init", "nnp_md_step", "nnp_get_state", "nnp_sync",
           "nnp_energy_forces_host", "nnp_md_step_host", "nnp_profile", "nnp_profile_read", "nnp_launch_count",
           "nnp_aev_len", "nnp_aev_active_columns", "nnp_aev_ladder", "nnp_md_set_langevin", "nnp_energy_forces_virial",
           "nnp_measure_peaks", "nnp_neighbors_no_alloc", "nnp_neighbors_no_alloc_error"]


class NnpError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__("%s: %s" % (STATUS_NAMES.get(status, status), msg))
        self.status = status


ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)      # void *(*alloc)(size_t bytes, void *user)
DEALLOC_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)          # void (*dealloc)(void *ptr, void *user)


class nnp_params(C.Structure):
    _fields_ = [
        ("n_species", C.c_int), ("rcr", C.c_float), ("rca", C.c_float),
        ("eta_r", C.c_float), ("n_shf_r", C.c_int), ("shf_r", C.POINTER(C.c_float)),
        ("eta_a", C.c_float), ("zeta", C.c_float), ("n_shf_a", C.c_int), ("shf_a", C.POINTER(C.c_float)),
        ("n_shf_z", C.c_int), ("shf_z", C.POINTER(C.c_float)),
        ("celu_alpha", C.c_float), ("n_nets", C.c_int), ("n_layers", C.c_int),
        ("widths", C.POINTER(C.c_int)), ("params", C.POINTER(C.c_float)),
        ("self_energy", C.POINTER(C.c_float)), ("mass", C.POINTER(C.c_float)),
        ("accel_conv", C.c_float), ("mm_mode", C.c_int), ("cap_r", C.c_int), ("cap_a", C.c_int),
        ("dense_aev", C.c_int),
        ("alloc", ALLOC_FN), ("dealloc", DEALLOC_FN), ("alloc_user", C.c_void_p),
    ]


_lib = None


def lib():
    """Loads libnnp_b200.so (built in-tree by paper_2405_01491_b200/build.py).  Fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("%s not found: run `python -m paper_2405_01491_b200.build` (nvcc, sm_100a)" % LIB_PATH)
        L = C.CDLL(LIB_PATH)
        vp, ip, fp, dp = C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p
        L.nnp_create.argtypes = [C.POINTER(vp), C.POINTER(nnp_params), C.c_int, C.c_int, C.c_int, vp]
        L.nnp_destroy.argtypes = [vp]
        L.nnp_destroy.restype = None
        L.nnp_last_error.argtypes = [vp]
        L.nnp_last_error.restype = C.c_char_p
        L.nnp_set_system.argtypes = [vp, C.c_int, ip, fp, C.POINTER(C.c_float), C.c_int, ip]
        L.nnp_set_system_cell.argtypes = [vp, C.c_int, ip, fp, C.POINTER(C.c_float), C.c_int, ip]
        L.nnp_set_positions.argtypes = [vp, fp]
        L.nnp_build_neighbors.argtypes = [vp, C.c_float]
        L.nnp_get_neighbors.argtypes = [vp, C.c_int, ip, ip, C.c_int]
        L.nnp_energy_forces.argtypes = [vp, dp, fp]
        L.nnp_get_aev.argtypes = [vp, fp]
        L.nnp_get_atomic_energies.argtypes = [vp, fp]
        L.nnp_md_init.argtypes = [vp, fp, C.c_float, C.c_float]
        L.nnp_md_step.argtypes = [vp, C.c_int]
        L.nnp_get_state.argtypes = [vp, fp, fp, dp, dp, ip]
        L.nnp_sync.argtypes = [vp]
        L.nnp_energy_forces_host.argtypes = [vp, C.c_int, ip, fp, C.POINTER(C.c_float), C.c_int, ip, C.c_float, dp, fp]
        L.nnp_md_step_host.argtypes = [vp, fp, fp, C.c_int, dp, dp]
        L.nnp_profile.argtypes = [vp, C.c_int]
        L.nnp_profile_read.argtypes = [vp, dp, ip]
        L.nnp_launch_count.argtypes = [vp]
        L.nnp_launch_count.restype = C.c_int64
        L.nnp_aev_len.argtypes = [vp]
        L.nnp_aev_active_columns.argtypes = [vp]
        L.nnp_aev_ladder.argtypes = [vp]
        L.nnp_md_set_langevin.argtypes = [vp, C.c_float, C.c_float, C.c_uint64]
        L.nnp_energy_forces_virial.argtypes = [vp, dp, fp, dp]
        L.nnp_measure_peaks.argtypes = [C.c_int, dp]
        L.nnp_neighbors_no_alloc.argtypes = [C.c_int, fp, C.POINTER(C.c_float), C.c_float, ip, ip, C.c_int, vp]
        L.nnp_neighbors_no_alloc_error.argtypes = []
        L.nnp_neighbors_no_alloc_error.restype = C.c_char_p
        _lib = L
    return _lib


def _ptr(t):
    """Address of a torch tensor / numpy array / None."""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        assert t.flags["C_CONTIGUOUS"]
        return t.ctypes.data
    assert t.is_contiguous()
    return t.data_ptr()


def _check(ctx, rc):
    if rc != NNP_OK:
        raise NnpError(rc, lib().nnp_last_error(ctx).decode())
    return rc


def make_params(consts, widths, params, mass, accel_conv, n_nets=1, self_energy=None, mm_mode=NNP_MM_FP32_SIMT,
                cap_r=0, cap_a=0, dense_aev=0, alloc=None, dealloc=None):
    """Fills an nnp_params from numpy arrays; returns (struct, keepalive list).  alloc / dealloc: Python callables
    (bytes, user) -> device pointer and (ptr, user) -> None, passed to the library as its device-memory hooks."""
    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    keep = dict(shf_r=f32(consts["shf_r"]), shf_a=f32(consts["shf_a"]), shf_z=f32(consts["shf_z"]),
                widths=np.ascontiguousarray(widths, dtype=np.int32), params=f32(params), mass=f32(mass),
                self_energy=None if self_energy is None else f32(self_energy))
    p = nnp_params()
    fp = lambda a: a.ctypes.data_as(C.POINTER(C.c_float))
    p.n_species = keep["widths"].shape[0]
    p.rcr, p.rca = float(consts["rcr"]), float(consts["rca"])
    p.eta_r, p.n_shf_r, p.shf_r = float(consts["eta_r"]), len(keep["shf_r"]), fp(keep["shf_r"])
    p.eta_a, p.zeta = float(consts["eta_a"]), float(consts["zeta"])
    p.n_shf_a, p.shf_a = len(keep["shf_a"]), fp(keep["shf_a"])
    p.n_shf_z, p.shf_z = len(keep["shf_z"]), fp(keep["shf_z"])
    p.celu_alpha = float(consts["celu_alpha"])
    p.n_nets, p.n_layers = int(n_nets), keep["widths"].shape[1] - 1
    p.widths = keep["widths"].ctypes.data_as(C.POINTER(C.c_int))
    p.params = fp(keep["params"])
    p.self_energy = fp(keep["self_energy"]) if keep["self_energy"] is not None else None
    p.mass = fp(keep["mass"])
    p.accel_conv, p.mm_mode, p.cap_r, p.cap_a = float(accel_conv), int(mm_mode), int(cap_r), int(cap_a)
    p.dense_aev = int(dense_aev)
    if alloc is not None:
        keep["alloc"], keep["dealloc"] = ALLOC_FN(alloc), DEALLOC_FN(dealloc)   # the thunks must outlive the context
        p.alloc, p.dealloc = keep["alloc"], keep["dealloc"]
    return p, keep


# ---- the C calls, one to one ------------------------------------------------------------------------
def nnp_create(params, max_atoms, max_mols=1, device=0, cuda_stream=0):
    ctx = C.c_void_p()
    rc = lib().nnp_create(C.byref(ctx), C.byref(params), int(max_atoms), int(max_mols), int(device),
                          C.c_void_p(int(cuda_stream)))
    if rc != NNP_OK:
        raise NnpError(rc, lib().nnp_last_error(None).decode())
    return ctx


def nnp_destroy(ctx):
    lib().nnp_destroy(ctx)


def nnp_last_error(ctx):
    return lib().nnp_last_error(ctx).decode()


def nnp_set_system(ctx, n_atoms, d_species, d_xyz, box, n_mols=1, d_mol_offsets=None):
    b = (C.c_float * 3)(*[float(x) for x in (box if box is not None else (0, 0, 0))])
    return _check(ctx, lib().nnp_set_system(ctx, int(n_atoms), _ptr(d_species), _ptr(d_xyz), b, int(n_mols),
                                            _ptr(d_mol_offsets)))


def nnp_set_system_cell(ctx, n_atoms, d_species, d_xyz, cell, n_mols=1, d_mol_offsets=None):
    """cell: 3 x 3, rows = lattice vectors (None: non-periodic)."""
    flat = [0.0] * 9 if cell is None else [float(x) for x in np.asarray(cell, dtype=np.float64).reshape(9)]
    h = (C.c_float * 9)(*flat)
    return _check(ctx, lib().nnp_set_system_cell(ctx, int(n_atoms), _ptr(d_species), _ptr(d_xyz), h, int(n_mols),
                                                 _ptr(d_mol_offsets)))


def nnp_set_positions(ctx, d_xyz):
    return _check(ctx, lib().nnp_set_positions(ctx, _ptr(d_xyz)))


def nnp_build_neighbors(ctx, skin=0.0):
    return _check(ctx, lib().nnp_build_neighbors(ctx, float(skin)))


def nnp_get_neighbors(ctx, which, d_counts, d_list, stride):
    return _check(ctx, lib().nnp_get_neighbors(ctx, int(which), _ptr(d_counts), _ptr(d_list), int(stride)))


def nnp_energy_forces(ctx, d_energy, d_forces):
    return _check(ctx, lib().nnp_energy_forces(ctx, _ptr(d_energy), _ptr(d_forces)))


def nnp_get_aev(ctx, d_aev):
    return _check(ctx, lib().nnp_get_aev(ctx, _ptr(d_aev)))


def nnp_get_atomic_energies(ctx, d_e_atom):
    return _check(ctx, lib().nnp_get_atomic_energies(ctx, _ptr(d_e_atom)))


def nnp_md_init(ctx, d_vel, dt_fs, skin):
    return _check(ctx, lib().nnp_md_init(ctx, _ptr(d_vel), float(dt_fs), float(skin)))


def nnp_md_step(ctx, n_steps):
    return _check(ctx, lib().nnp_md_step(ctx, int(n_steps)))


def nnp_get_state(ctx, d_xyz=None, d_vel=None, d_epot=None, d_ekin=None, d_n_rebuilds=None):
    return _check(ctx, lib().nnp_get_state(ctx, _ptr(d_xyz), _ptr(d_vel), _ptr(d_epot), _ptr(d_ekin), _ptr(d_n_rebuilds)))


def nnp_sync(ctx):
    return _check(ctx, lib().nnp_sync(ctx))


def nnp_energy_forces_host(ctx, n_atoms, h_species, h_xyz, box, n_mols, h_mol_offsets, skin, h_energy, h_forces):
    b = (C.c_float * 3)(*[float(x) for x in (box if box is not None else (0, 0, 0))])
    return _check(ctx, lib().nnp_energy_forces_host(ctx, int(n_atoms), _ptr(h_species), _ptr(h_xyz), b, int(n_mols),
                                                    _ptr(h_mol_offsets), float(skin), _ptr(h_energy), _ptr(h_forces)))


def nnp_md_step_host(ctx, h_xyz, h_vel, n_steps, h_epot, h_ekin):
    return _check(ctx, lib().nnp_md_step_host(ctx, _ptr(h_xyz), _ptr(h_vel), int(n_steps), _ptr(h_epot), _ptr(h_ekin)))


NNP_N_STAGES = 13
STAGE_NAMES = ["kick_drift", "neighbor_build", "aev_forward", "mlp_fwd_l1", "mlp_fwd_l2", "mlp_fwd_l3_out",
               "mlp_bwd_l3", "mlp_bwd_l2", "mlp_bwd_l1_dEdG", "energy_sum", "aev_backward_scatter", "kick_ekin",
               "mlp_fused_chain"]


def nnp_profile(ctx, stride):
    return _check(ctx, lib().nnp_profile(ctx, int(stride)))


def nnp_profile_read(ctx):
    ms = np.zeros(NNP_N_STAGES, dtype=np.float64)
    cnt = np.zeros(NNP_N_STAGES, dtype=np.int64)
    _check(ctx, lib().nnp_profile_read(ctx, _ptr(ms), _ptr(cnt)))
    return ms, cnt


def nnp_launch_count(ctx):
    return int(lib().nnp_launch_count(ctx))


def nnp_aev_len(ctx):
    return int(lib().nnp_aev_len(ctx))


def nnp_aev_active_columns(ctx):
    return int(lib().nnp_aev_active_columns(ctx))


def nnp_aev_ladder(ctx):
    return int(lib().nnp_aev_ladder(ctx))


def nnp_md_set_langevin(ctx, gamma, kT, seed):
    return _check(ctx, lib().nnp_md_set_langevin(ctx, float(gamma), float(kT), int(seed)))


def nnp_energy_forces_virial(ctx, d_energy, d_forces, d_virial):
    return _check(ctx, lib().nnp_energy_forces_virial(ctx, _ptr(d_energy), _ptr(d_forces), _ptr(d_virial)))


NNP_N_PEAKS = 13
PEAK_NAMES = ["fp32_fma_tflops", "mufu_ex2_gops", "tf32_tcgen05_ss_tflops", "tf32_tcgen05_ts_tflops",
              "cycles_per_mma_m128n256k8_ss", "cycles_per_mma_m128n256k8_ts"] + \
             ["cycles_per_mma_m128n%dk8_ts_sweep" % n for n in range(64, 257, 32)]


def nnp_measure_peaks(device=0):
    """Measured roofline denominators of `device` (include/nnp.h), as a dict."""
    out = np.zeros(NNP_N_PEAKS, dtype=np.float64)
    rc = lib().nnp_measure_peaks(int(device), _ptr(out))
    if rc != NNP_OK:
        raise RuntimeError("nnp_measure_peaks failed with status %d" % rc)
    return dict(zip(PEAK_NAMES, (float(v) for v in out)))


NNP_NO_ALLOC_MAX_ATOMS = 16384


def nnp_neighbors_no_alloc_error():
    return (lib().nnp_neighbors_no_alloc_error() or b"").decode()


def nnp_neighbors_no_alloc(n_atoms, d_xyz, box, rcut, d_counts, d_list, stride, stream=None):
    """Neighbour lists of one point set with the scratch memory in the library's static device array (include/nnp.h):
    no ctx, no allocation, no synchronisation.  box: 3 edge lengths or None (not periodic)."""
    b = None if box is None else (C.c_float * 3)(*[float(x) for x in box])
    rc = lib().nnp_neighbors_no_alloc(int(n_atoms), _ptr(d_xyz), b, float(rcut), _ptr(d_counts), _ptr(d_list), int(stride),
                                      stream)
    if rc != NNP_OK:
        raise NnpError(rc, nnp_neighbors_no_alloc_error())
    return rc
