/*
 * nnp.h -- C-ABI of the B200-native ANI-2x energy / force / MD hot path.
 *
 * What is computed (citations are /root/reference/PAPER.md lines + SURVEY.md 8(c) items, restated in
 * DESIGN.md "The path"): one ANI-like evaluation as in Fig. 2 of the FeNNol paper:
 *   stage 1  neighbour lists (GraphGenerator / GraphFilter, L41-55; cell list + Verlet skin, L49, L341)
 *   stage 2  atomic environment vectors (ANI_AEV, L71, L79, cosine switch L61, angular form L443)
 *   stage 3  species-specialised MLPs (ChemicalNet, L87) summed per structure (L176)
 *   stage 4  forces = -dE/dx, the hand-written reverse pass of what the paper gets from jax.grad (L65, L176)
 *   stage 5  velocity Verlet, GPU-resident (fennol_md NVE, L307)
 *
 * Conventions
 *   - Every function returns NNP_OK (0) or a negative nnp_status; none throws or exits.  After a failure
 *     nnp_last_error(ctx) returns a static / ctx-owned description.
 *   - Pointer names say where the memory lives: d_* device memory owned by the caller (e.g. a torch
 *     tensor) that must stay valid until the stream work that uses it has completed; h_* host memory
 *     (pinned memory makes the copies asynchronous).  The library never frees caller memory.
 *   - All work is enqueued on the CUDA stream given to nnp_create and the calls return without waiting,
 *     except where "synchronises" is stated.  Conditions only visible on the device (neighbour capacity
 *     overflow) are latched in a device flag and reported by the next synchronising call.
 *   - Atom indices in and out are the caller's original order.  Internally atoms are kept sorted by
 *     (species, cell); that order is never visible.
 *   - Units: Angstrom, fs, amu, energy unit of the weights (kcal/mol in the tests); accelerations are
 *     accel_conv * F / m.
 *   - Arithmetic: fp32 throughout, energies accumulated in fp64.  The MLP contractions run in the mode
 *     chosen by mm_mode and the mode is part of every reported number.
 *
 * Fixed shape of this build (nnp_create returns NNP_EINVAL otherwise): n_species <= 7, n_shf_r == 16,
 * n_shf_a == 8, n_shf_z == 4, n_layers == 4 with widths[s] = {1008-compatible AEV length, h1, h2, h3, 1},
 * hidden widths multiples of 32 and <= 256.
 */
#ifndef NNP_H
#define NNP_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct nnp_ctx nnp_ctx; /* opaque; owned by the library; freed by nnp_destroy */

typedef enum {
    NNP_OK = 0,
    NNP_EINVAL = -1,    /* bad argument / unsupported shape */
    NNP_ENOMEM = -2,    /* device or host allocation failed */
    NNP_ECUDA = -3,     /* CUDA runtime error (message in nnp_last_error) */
    NNP_ECAPACITY = -4, /* a neighbour row exceeded cap_r / cap_a: recreate with larger caps */
    NNP_ESTALE = -5,    /* energy/forces or MD requested without a neighbour list for the current system */
    NNP_EBOX = -6,      /* periodic box edge < 2*(cutoff+skin): minimum image not unique (reading C1) */
    NNP_ERANGE = -7     /* mm_mode 4: an activation left the range of the scaled fp16 split (|value| > 3750): the result
                           of this evaluation is invalid; use mm_mode 1 for such a model */
} nnp_status;

/* How the MLP contractions are computed (Fig. 3: matmul precision decides energy conservation):
 * 0 fp32 FMA on the CUDA cores; 1 (default of the tests and the bench) 3xTF32 on tcgen05, fp32-grade; 2 plain TF32 on
 * tcgen05 (fails the parity bars, kept for the precision study); 3 fp32 operands with every product and sum in fp64
 * (DFMA on the CUDA cores) -- the fp64 leg of the precision study, slow; 4 "3xF16": all six GEMMs of every network and
 * species as ONE fused tcgen05 kernel with every fp32 operand split into fp16 hi + fp16 lo (11 + 11 significant bits as in
 * mode 1, power-of-two scaling against fp16's exponent range, fp32 accumulation), fp32-grade; models the chain does not take
 * (a hidden width outside [64, 256], more than 64 (network, species) pairs) run as in mode 1.  Out-of-range activations ->
 * NNP_ERANGE. */
enum { NNP_MM_FP32_SIMT = 0, NNP_MM_3XTF32_TC = 1, NNP_MM_TF32_TC = 2, NNP_MM_FP64_SIMT = 3, NNP_MM_3XF16_TC = 4 };

typedef struct {
    int n_species;            /* <= 7; ANI-2x: 7, index order H,C,N,O,S,F,Cl (reading B2) */
    float rcr, rca;           /* radial / angular cutoffs, Angstrom (5.1 / 3.5; reading A1) */
    float eta_r;              /* radial Gaussian exponent */
    int n_shf_r;              /* 16 */
    const float *shf_r;       /* host [n_shf_r] */
    float eta_a, zeta;        /* angular Gaussian exponent, angular power */
    int n_shf_a;              /* 8 */
    const float *shf_a;       /* host [n_shf_a] */
    int n_shf_z;              /* 4 */
    const float *shf_z;       /* host [n_shf_z], radians */
    float celu_alpha;         /* CELU alpha (0.1) */
    int n_nets;               /* ensemble size; energies and forces are the arithmetic mean (reading B5) */
    int n_layers;             /* 4 affine layers */
    const int *widths;        /* host [n_species][n_layers+1], widths[s][0] = AEV length, widths[s][4] = 1 */
    const float *params;      /* host, flat: for net, for species, for layer: W[in][out] row-major then b[out] */
    const float *self_energy; /* host [n_species] or NULL (= 0); added per atom, no force (reading B4) */
    const float *mass;        /* host [n_species], amu */
    float accel_conv;         /* a = accel_conv * F / m  (4.184e-4 for kcal/mol, A, fs, amu; reading B6) */
    int mm_mode;              /* NNP_MM_*: how the MLP contractions are computed */
    int cap_r, cap_a;         /* capacities of the radial / angular neighbour ROWS (entries with r < cutoff + skin); 0 =>
                                 160 / 64; multiples of 4 in [4, 65532].  Independently of cap_a, a centre may have at most
                                 64 angular neighbours INSIDE the cutoff rca (the AEV kernels keep them in shared memory);
                                 any overflow is reported as NNP_ECAPACITY, never truncated silently. */
    int dense_aev;            /* 0 (default): AEV columns of species absent from the loaded system -- identically zero
                                 for every atom -- are neither stored nor multiplied (the layer-1 weights are gathered
                                 to the active columns at nnp_set_system; results are unchanged).  1: always keep all
                                 aev_len columns (e.g. 1008), as a plain implementation would. */
    /* Device-memory hooks (north_star: PyTorch supplies device memory): every device buffer the library
     * owns is obtained from alloc(bytes, alloc_user) -- which returns a device pointer aligned to >= 256 bytes on the
     * device given to nnp_create, or NULL on failure (-> NNP_ENOMEM) -- and returned with dealloc(ptr, alloc_user), at
     * nnp_destroy at the latest.  E.g. torch.cuda.caching_allocator_alloc / _delete.  Both NULL: cudaMalloc / cudaFree. */
    void *(*alloc)(size_t bytes, void *alloc_user);
    void (*dealloc)(void *ptr, void *alloc_user);
    void *alloc_user;
} nnp_params;

/* The model of PAPER.md L176 (Fig. 2: AEV embedding, species-specialised networks, sum) with the constants of
 * DESIGN.md section 2 as parameters.  Copies all parameters to the device (the caller keeps its arrays) and allocates
 * every scratch buffer (through nnp_params.alloc if given) for up to max_atoms atoms in up to max_mols structures.  cuda_stream is a cudaStream_t (NULL = legacy
 * default stream).  Synchronises. */
int nnp_create(nnp_ctx **out, const nnp_params *p, int max_atoms, int max_mols, int device, void *cuda_stream);
void nnp_destroy(nnp_ctx *ctx);
const char *nnp_last_error(const nnp_ctx *ctx); /* ctx may be NULL (create failures) */

/* Loads a system: species index per atom (0..n_species-1) and coordinates [n][3] (fp32, Angstrom, need
 * not be wrapped).  h_box: orthorhombic edge lengths; all zero => non-periodic.  Batches (PAPER.md L41,
 * L176): d_mol_offsets[n_mols+1] gives each structure's atom range in the concatenated arrays, atoms of
 * different structures never interact; NULL => one structure.  With a box, a batch is a set of replicas of ONE
 * periodic cell (same edge lengths for all, e.g. the beads of a ring polymer): every structure gets
 * its own set of cell-list bins; energies come back per structure.  (MD and the virial take one structure.)
 * Invalidates neighbour lists and MD state.  Synchronises (species counts are read back). */
int nnp_set_system(nnp_ctx *ctx, int n_atoms, const int32_t *d_species, const float *d_xyz,
                   const float h_box[3], int n_mols, const int32_t *d_mol_offsets);

/* The same with a GENERAL cell ("optionally cell vectors", L49, L307 "minimum image or
 * all images"): h_cell[9] (host), rows = the lattice vectors a, b, c in Angstrom, any orientation, triclinic allowed; NULL or
 * all zero = non-periodic.  Atoms interact with ALL periodic images inside the cutoffs:
 *   - every perpendicular width of the cell >= 2 (rcr + 0.5 A): minimum image, found by rounding the displacement's
 *     fractional coordinates (a diagonal cell takes exactly the orthorhombic path of nnp_set_system);
 *   - a narrower cell (down to cells smaller than the cutoff, where an atom sees several images of the same neighbour and
 *     of itself) is evaluated, exactly, as the smallest m0 x m1 x m2 supercell that reaches that width: the library holds
 *     n_atoms * m0 m1 m2 internal atoms (this product must be <= max_atoms, else NNP_EBOX), returns energy / virial per
 *     cell and the forces, AEVs, neighbour rows (an image of atom j is reported as j) of the caller's atoms.  One
 *     structure only.  In MD the copies are reset to their atom's state (+ the copy's lattice shift) after every drift
 *     and before every kick, so the supercell stays exactly periodic in the caller's cell.
 * nnp_build_neighbors returns NNP_EBOX if a width of the (super)cell is below 2 (rcr + skin). */
int nnp_set_system_cell(nnp_ctx *ctx, int n_atoms, const int32_t *d_species, const float *d_xyz, const float h_cell[9],
                        int n_mols, const int32_t *d_mol_offsets);

/* Replaces the coordinates of the loaded system ([n][3], original order); lists stay as they are (the
 * caller asserts no atom moved more than skin/2 since nnp_build_neighbors). */
int nnp_set_positions(nnp_ctx *ctx, const float *d_xyz);

/* Stage 1.  Builds the directed radial list {j : r_ij < rcr+skin} and angular list {j : r_ij < rca+skin}
 * (same structure only, minimum image) with an O(N) cell list; membership is the fp32 predicate of
 * reading A3.  Re-sorts the internal atom order.  Returns NNP_EBOX if a periodic edge is
 * shorter than 2*(rcr+skin). */
int nnp_build_neighbors(nnp_ctx *ctx, float skin);

/* Test hook: rows of list `which` (0 radial, 1 angular) with ORIGINAL atom indices, row i for original
 * atom i, unsorted.  d_counts[n]; d_list[n][stride], entries beyond counts[i] untouched.  Synchronises;
 * reports NNP_ECAPACITY. */
int nnp_get_neighbors(nnp_ctx *ctx, int which, int32_t *d_counts, int32_t *d_list, int stride);

/* Stages 2-4 with the current lists.  d_energy[n_mols] fp64 (mean over nets, + self energies);
 * d_forces[n][3] fp32 in original order, may be NULL (energy only still runs the full path). */
int nnp_energy_forces(nnp_ctx *ctx, double *d_energy, float *d_forces);

/* Energy, forces and the virial of ONE structure (n_mols = 1; PAPER.md L262 energy_and_forces_and_virial, SURVEY.md
 * 8(f) item 2; any cell of nnp_set_system / nnp_set_system_cell): d_virial[9] fp64, row-major V_ab = dE/d eps_ab = sum over every displacement
 * vector d the energy is built from of d_a (dE/dd)_b -- the derivative of the energy under the homogeneous
 * deformation x -> (1 + eps) x, cell -> (1 + eps) cell; symmetric; stress = V / volume; without a cell
 * V_ab = -sum_i x_ia F_ib.  Accumulated in fp32 per lane and in fp64 across warps by the reverse AEV kernel.
 * NNP_EINVAL for batched structures.  Otherwise as nnp_energy_forces. */
int nnp_energy_forces_virial(nnp_ctx *ctx, double *d_energy, float *d_forces, double *d_virial);

/* Test hooks (valid after nnp_energy_forces): AEVs [n][aev_len] and per-atom energies [n], original order. */
int nnp_get_aev(nnp_ctx *ctx, float *d_aev);
int nnp_get_atomic_energies(nnp_ctx *ctx, float *d_e_atom);

/* Stage 5.  nnp_md_init: velocities [n][3] (A/fs, original order), time step (fs), Verlet skin (A);
 * builds the lists and evaluates the initial forces.  nnp_md_step: n_steps of velocity Verlet
 * (v += dt/2 a; x += dt v; rebuild lists iff max_i |x_i - x_i(last build)| > skin/2, decided on the
 * device; forces; v += dt/2 a), no host synchronisation inside (reading C2).
 * Batches (n_mols > 1: molecules, or replicas of one periodic cell - the ring-polymer beads of PAPER.md L309 get their
 * potential energies and forces this way): every structure takes the same steps independently of the others; the rebuild
 * test is one flag for the whole batch (any atom of any structure beyond skin/2 rebuilds all lists).  The bead-bead springs
 * of a ring-polymer Hamiltonian are not part of this library. */
int nnp_md_init(nnp_ctx *ctx, const float *d_vel, float dt_fs, float skin);
int nnp_md_step(nnp_ctx *ctx, int n_steps);

/* Langevin dynamics with the BAOAB splitting ("Langevin dynamics (using the BAOAB scheme)", the
 * setting of the paper's benchmarks, L323).  After nnp_md_init; from then on nnp_md_step does
 *   v += dt/2 a;  x += dt/2 v;  v = c1 v + c2_s xi;  x += dt/2 v;  [rebuild test]  forces;  v += dt/2 a
 * with c1 = exp(-gamma dt), c2_s = sqrt((1 - c1^2) kT accel_conv / m_s), xi three standard normals per atom and step
 * from Philox4x32-10 with counter (original atom index, step since nnp_md_init, 0, 0) and key = seed (uniforms
 * ((r >> 9) + 1/2) 2^-23, Box-Muller), so a trajectory does not depend on how the steps are split over calls.
 * gamma [1/fs] = 0 switches back to velocity Verlet.  kT in energy units.  nnp_md_init resets to velocity Verlet. */
int nnp_md_set_langevin(nnp_ctx *ctx, float gamma, float kT, uint64_t seed);

/* Copies out the current state in original order; any pointer may be NULL.  d_epot/d_ekin: fp64 [n_mols]
 * (per structure: potential energy of the last force evaluation, kinetic energy after the last step, energy units);
 * d_n_rebuilds: list builds since nnp_md_init (the initial one included).  Asynchronous. */
int nnp_get_state(nnp_ctx *ctx, float *d_xyz, float *d_vel, double *d_epot, double *d_ekin, int32_t *d_n_rebuilds);

/* Waits for the stream and reports latched device conditions (NNP_ECAPACITY, NNP_ECUDA). */
int nnp_sync(nnp_ctx *ctx);

/* Host-buffer entry points (the end-to-end path: H2D copies, the same kernels, D2H copies; synchronise).
 * nnp_energy_forces_host = nnp_set_system + nnp_build_neighbors(skin) + nnp_energy_forces.
 * nnp_md_step_host: uploads h_xyz/h_vel [n][3] into the running MD state (atoms as in nnp_set_system; lists
 * are kept and rebuilt by the displacement rule), runs n_steps, downloads positions, velocities, epot, ekin (the two
 * scalars and the device-side error flags travel in one 40-byte pinned copy).  Synchronises before returning.
 * h_xyz / h_vel must be the state returned by the previous call (or the state given to nnp_md_init), possibly with atoms
 * shifted by whole cell vectors: the first half kick uses the forces of the previous evaluation, which are NOT recomputed
 * from the uploaded positions. */
int nnp_energy_forces_host(nnp_ctx *ctx, int n_atoms, const int32_t *h_species, const float *h_xyz,
                           const float h_box[3], int n_mols, const int32_t *h_mol_offsets, float skin,
                           double *h_energy, float *h_forces);
int nnp_md_step_host(nnp_ctx *ctx, float *h_xyz, float *h_vel, int n_steps, double *h_epot, double *h_ekin);

/* Per-stage device timing for the bench (CUDA events on the ctx stream around the stage launches of every
 * `stride`-th nnp_md_step step / nnp_energy_forces call; stride 0 switches it off and clears the sums).
 * nnp_profile_read synchronises and returns, per stage, the summed milliseconds and the number of samples:
 * 0 kick+drift, 1 neighbour build (all its kernels; near zero on steps without a rebuild), 2 AEV forward,
 * 3..5 MLP forward layers 1..3 (layer 3 includes the output layer), 6..8 MLP reverse layers 3..1 (8 = dE/dG),
 * 9 energy sum, 10 AEV reverse + force scatter, 11 kick + kinetic energy, 12 the fused MLP chain of mm_mode 4 (all six
 * GEMMs in one launch; stages 3..8 stay zero then).
 * Arrays of NNP_N_STAGES entries. */
#define NNP_N_STAGES 13
int nnp_profile(nnp_ctx *ctx, int stride);
int nnp_profile_read(nnp_ctx *ctx, double *h_ms_sum, int64_t *h_samples);

/* Introspection for the bench: number of kernel launches issued by this ctx so far. */
int64_t nnp_launch_count(const nnp_ctx *ctx);
int nnp_aev_len(const nnp_ctx *ctx);            /* full AEV length of the model (1008 for 7 species) */
int nnp_aev_active_columns(const nnp_ctx *ctx); /* columns stored for the loaded system (see nnp_params.dense_aev) */
/* 1 if the AEV kernels evaluate the Gaussian shift sets by the ladder recurrence (uniformly spaced ShfR / ShfA whose
 * powers stay in fp32 range), 0 if every exponential is evaluated directly (any shift set; NNP_NO_LADDER=1 in the
 * environment at nnp_create forces this).  Same results within the parity tolerances either way. */
int nnp_aev_ladder(const nnp_ctx *ctx);

/* Roofline denominators measured on `device` (the TF32 tcgen05, fp32 FMA and SFU peaks are to be
 * micro-benchmarked by the builder).  Runs three register/shared-memory-resident micro-kernels on every SM, best of a few
 * launches each, synchronously on the default stream, and fills h_out (host, NNP_N_PEAKS doubles):
 *   0 fp32 FMA TFLOP/s (2 flops per FMA), 1 MUFU ex2 G ops/s, 2 dense TF32 tcgen05.mma TFLOP/s with both operands in
 *   shared memory, 3 the same with A in tensor memory (the operand form of the MLP GEMMs), 4 / 5 SM cycles per
 *   M128 N256 K8 MMA instruction for the two forms, 6..12 SM cycles per M128 N K8 instruction (A in tensor memory) for
 *   N = 64, 96, 128, 160, 192, 224, 256.  Needs no ctx; allocates and frees a few KB.  Diagnostic only:
 * nothing on the energy/force/MD path calls it.  Returns NNP_OK, NNP_EINVAL (null), NNP_ECUDA, NNP_ENOMEM. */
#define NNP_N_PEAKS 13
int nnp_measure_peaks(int device, double *h_out);

/* Neighbour lists without any allocation (csrc/no_alloc.cu), for callers that cannot call cudaMalloc: code under CUDA graph
 * capture, tight serving loops, harnesses that forbid it.  The cell-list build of stage 1 for ONE point
 * set: for every atom i the set {j != i : r_ij < rcut} under the minimum image of an orthorhombic box, membership decided by
 * the same fp32 predicate as nnp_build_neighbors (reading A3) - the rows equal those of nnp_get_neighbors for the
 * same radius.  Needs no ctx, calls no cudaMalloc / cudaFree and no allocating library routine, does not synchronise: it
 * enqueues one memset and four kernels on `cuda_stream` (a cudaStream_t, NULL = default stream) of the CURRENT device.
 *   n_atoms   <= NNP_NO_ALLOC_MAX_ATOMS (else NNP_EINVAL, message in nnp_neighbors_no_alloc_error()); 0 is a no-op
 *   d_xyz     device, [n_atoms][3] fp32, any image of the atoms (wrapped internally)
 *   h_box     host, 3 edge lengths; NULL or all zero: not periodic (all pairs are tested).  NNP_EBOX if an edge < 2 rcut
 *   d_counts  device, [n_atoms] int32: number of neighbours of atom i (the full count, also where it exceeds `stride`)
 *   d_list    device, [n_atoms][stride] int32: the neighbours of atom i, unsorted; entries beyond min(count, stride) untouched
 * All buffers are the caller's; nothing is retained.  The scratch memory (positions as float4, cell keys, the order by
 * cell, the cell histogram and start table: ~450 KiB) is ONE array in the library image, held by every GPU that loads the
 * library until the process exits, and shared by all calls: calls that overlap on one GPU (two streams, concurrent graph
 * launches) race on it - serialise them.  The first call on a device looks up the array's device address
 * (cudaGetSymbolAddress): make that call outside a stream capture. */
#define NNP_NO_ALLOC_MAX_ATOMS 16384
int nnp_neighbors_no_alloc(int n_atoms, const float *d_xyz, const float h_box[3], float rcut, int32_t *d_counts,
                           int32_t *d_list, int stride, void *cuda_stream);
const char *nnp_neighbors_no_alloc_error(void); /* message of the calling thread's last failed nnp_neighbors_no_alloc */

#ifdef __cplusplus
}
#endif
#endif /* NNP_H */
