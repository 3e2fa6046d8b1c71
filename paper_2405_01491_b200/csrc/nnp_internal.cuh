// Internal declarations of the CUDA path (sm_100a).  Not part of the C-ABI (include/nnp.h).
// Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "../../include/nnp.h"

#define NNP_MAX_SPECIES 8
#define NNP_MAX_GROUPS 16  // (network, species) groups of one grouped GEMM launch: ensembles batch their networks per layer
#define NNP_NSHF_R 16
#define NNP_NSHF_A 8
#define NNP_NSHF_Z 4
#define NNP_ANG_BLOCK (NNP_NSHF_A * NNP_NSHF_Z) /* 32 features per species pair */
#define NNP_NLAYERS 4
#define NNP_AEV_SCHED_LEN 1056 /* per AEV kernel: [0] exit counter, [32 + s] tickets of SM range s (s < 1024) */
#define NNP_TRI_LEN 2016 /* pairs (lo < hi) with hi < 64: decode table of the AEV kernels */

// Device error flags latched by kernels, reported by synchronising calls.
enum { NNP_FLAG_CAP_R = 1, NNP_FLAG_CAP_A = 2, NNP_FLAG_RANGE = 4 };

// ---- periodic cell grid / molecule bins (stage 1) ------------------------------------------------
struct GridInfo {
    int nc[3];        // cells per dimension (periodic) or {n_mols,1,1} (batched molecules)
    int ncell;        // bins in all: nc[0]*nc[1]*nc[2] x (structures sharing the box), or n_mols
    int ncell_box;    // periodic: nc[0]*nc[1]*nc[2], the bins of ONE structure (replica r owns bins [r, r+1) * ncell_box)
    int periodic;     // 1: orthorhombic minimum image; 0: bins are molecules
    float box[3];
    float inv_box[3]; // 1.0f / box (IEEE division on the host)
    float cell_scale[3]; // nc / box
    // general (triclinic) cell: rows of h are the lattice vectors, frac_c(x) = hinv[3c..3c+2] . x; bins are
    // cut in fractional coordinates.  tric = 0: the orthorhombic arithmetic above (reading A3) is used unchanged.
    int tric;
    float h[9], hinv[9];
};

// ---- AEV constants (stage 2/4), passed to kernels by value --------------------------------------
// Columns of G: only the feature blocks of species PRESENT in the loaded system are stored ("active columns":
// np*16 radial + np(np+1)/2*32 angular); blocks of absent species are identically zero for every atom, so
// dropping them (and the matching rows of the layer-1 weights) changes no result.  cmap/plist translate between
// model species and the compact index; with dense_aev (or all species present) the layout is the full one.
struct AevParams {
    int S;           // species of the model
    int np;          // species present in the loaded system (compact index 0..np-1, ascending species)
    int cmap[NNP_MAX_SPECIES];  // species -> compact index, -1 if absent
    int plist[NNP_MAX_SPECIES]; // compact index -> species
    int n_rad;       // np*16
    int aev_len;     // n_rad + np(np+1)/2*32 (active columns)
    int kpad;        // row stride of G / dG in floats (aev_len rounded up to 32)
    int cap_r, cap_a;
    float rcr, rca;
    float rcr2, rca2;
    float pi_rcr, pi_rca;      // pi / cutoff
    float neg_eta_r_log2e;     // -eta_r * log2(e)
    float neg_eta_a_log2e;
    float eta_r, eta_a, zeta;
    float shf_r[NNP_NSHF_R];
    float shf_a[NNP_NSHF_A];
    float cos_z[NNP_NSHF_Z], sin_z[NNP_NSHF_Z];
    float ka;                   // sqrt(eta_a log2 e): exp(-eta_a u^2) = 2^-(ka u)^2
    float ka_shf[NNP_NSHF_A];   // ka * shf_a
    float kr;                   // sqrt(eta_r log2 e)
    float kr_shf[NNP_NSHF_R];   // kr * shf_r
    // Gaussian ladder (aev.cu): with uniformly spaced shifts, exp(-eta (r - Shf_k)^2) for the four shifts k = 4m + J
    // of a group follows from the anchor k = 4m + 1 by powers of Q = 2^(2 delta w_0): e_k = lad_c[k] e_anchor Q^(J-1),
    // w_0 = k_ (r - Shf_1), delta = k_ (Shf_1 - Shf_0).  6 (radial) / 4 (angular) exponentials instead of 16 / 8.
    int ladder;                 // 1: both shift sets are uniform and the powers stay inside fp32 range
    float dlt_r, dlt_a;         // delta (scaled shift spacing)
    float lad_r[NNP_NSHF_R];    // constant factors of the deferred scaling, 1 without ladder
    float lad_a[NNP_NSHF_A];
    int periodic;
    float box[3], inv_box[3];
    int tric;                  // general cell: minimum image by rounding the fractional displacement (hinv), then h
    float h[9], hinv[9];
    // Derived constants of the inner loops, computed once on the host (nnp_aev_derive): the kernels take them straight
    // from the parameter bank (the pairs as one 64-bit uniform-register operand of the packed f32x2 instructions)
    // instead of re-deriving them per loop trip under register pressure.
    float2 hcz2[NNP_NSHF_Z / 2], hsz2[NNP_NSHF_Z / 2], nhsz2[NNP_NSHF_Z / 2]; // 1/2 cos ShfZ, 1/2 sin ShfZ, -1/2 sin ShfZ
    float2 nka_shf2[NNP_NSHF_A / 2];  // -ka_shf, pairs (2a, 2a+1)
    float2 nkr_shf2[NNP_NSHF_R / 2];  // -kr_shf, pairs (2k, 2k+1)
    float2 nkr_anc2[NNP_NSHF_R / 8];  // ladder anchors (-kr_shf[8m+1], -kr_shf[8m+5])
    float2 nka_anc2;                  // (-ka_shf[1], -ka_shf[5])
    float half_ka;                    // ka / 2: ka (r_ij + r_ik) / 2
    float k_ang0;                     // zeta * 0.95 (d base^zeta / d cos theta, with the 1/2 of the base folded in)
    float zm1;                        // zeta - 1
    float half_drb_scale;             // (1/2) (-2 eta_a / ka)
    float dr_scale;                   // -2 eta_r / kr
    float nh_pi_rcr, nh_pi_rca;       // -(1/2) pi / cutoff: fc' = nh_pi_rc sin(pi r / rc)
    float two_dlt_r, two_dlt_a;
};
void nnp_aev_derive(AevParams &a);

// ---- grouped GEMM description (stage 3/4) --------------------------------------------------------
enum GemmEpilogue {
    EPI_CELU = 0,     // C = celu(acc + bias)
    EPI_CELU_OUT = 1, // h = celu(acc + bias); e_atom[m] += sum_n h*w4[n]; C = w4[n] * celu'(h)
    EPI_DCELU = 2,    // C = acc * celu'(H) with H read from C (in place)
    EPI_STORE = 3,    // C = acc
    EPI_ACCUM = 4,    // C += acc
    EPI_RED = 5       // C += acc with vector reductions in memory (several groups of one launch add into the same rows;
                      // tensor-core path only)
};

struct GemmGroup {
    const float *A;   // [M][lda]   K-contiguous rows
    const float *B;   // [K][N]     row-major (SIMT path)
    const float *Bt;  // [N][K]     K-contiguous rows (tensor-core path, plain TF32 rounds it on the fly)
    const float *Bt_hi, *Bt_lo; // tf32 hi / lo split of Bt (3xTF32; nullptr in SIMT mode)
    float *C;         // [M][ldc]
    const float *bias; // [N] or nullptr
    const float *w4;  // [N] last-layer weights (EPI_CELU_OUT)
    float *e_atom;    // [M] (EPI_CELU_OUT)
    int M, N, K, lda, ldc;
};

struct GemmBatch {
    GemmGroup g[NNP_MAX_GROUPS];
    int n_groups;
    int tile_off[NNP_MAX_GROUPS + 1]; // prefix sum of M tiles per group (tile height given at launch)
    float alpha;                       // CELU alpha
};

// ---- context -----------------------------------------------------------------------------------
struct LayerW {
    float *W;  // device [in_pad][out]
    float *Wt; // device [out][in_pad]
    float *b;  // device [out]
    float *W_hi, *W_lo, *Wt_hi, *Wt_lo; // tf32 splits (tensor-core modes only)
    int in, in_pad, out;
    float wmax; // max |w| (scaling of the fp16 split, mlp_fused.cu)
};
// layer 1 restricted to the active columns of the loaded system (built by nnp_set_system)
struct Layer1C {
    float *W, *Wt, *W_hi, *W_lo, *Wt_hi, *Wt_lo; // [kpad][out] / [out][kpad]
};

struct nnp_fused; // mlp_fused.cu: packed weight tiles, group table and tile ranges of the fused MLP kernel

struct nnp_ctx {
    // model
    int S, n_nets, mm_mode, dense_aev;
    int tc_mode;                    // mm_mode is one of the tcgen05 modes (weights carry tf32 hi / lo splits)
    int split3;                     // unfused tcgen05 GEMMs run 3xTF32 (modes 1 and 4), else plain TF32
    int aev_len_full, kpad_full;    // 1008 / 1024 for 7 species
    unsigned present_mask;          // species mask the compact layer-1 copies were built for (0: none yet)
    Layer1C *l1c;                   // host array [n_nets][S]
    float *d_l1c_blob;              // device storage of the compact layer-1 copies (sized for the full layout)
    int *d_fmap;                    // [kpad_full] compact column -> full column (-1: zero padding)
    uint16_t *d_tri;                // [NNP_TRI_LEN] pair decode table (aev.cu)
    int widths[NNP_MAX_SPECIES][NNP_NLAYERS + 1];
    int hmax[3]; // max hidden widths over species (strides of the activation buffers)
    AevParams aev;
    float alpha, accel_conv;
    float mass[NNP_MAX_SPECIES];
    float e_shift[NNP_MAX_SPECIES]; // mean over nets of last-layer bias + self energy
    LayerW *layers;                 // host array [n_nets][S][4]
    float *d_params_blob;           // all device weights in one allocation
    float *d_inv_mass_conv;         // [S] accel_conv / mass
    float *d_mass;                  // [S]
    float *d_e_shift;               // [S]

    cudaStream_t stream;
    // device-memory hooks of nnp_params (nullptr: cudaMalloc / cudaFree)
    void *(*alloc_fn)(size_t, void *);
    void (*dealloc_fn)(void *, void *);
    void *alloc_user;
    int device, max_atoms, max_mols;
    int64_t launches;
    std::string err;
    // per-stage event timing (nnp_profile)
    int prof_stride, prof_active;
    int64_t prof_calls;
    std::vector<cudaEvent_t> prof_pool;          // recycled events
    std::vector<std::pair<cudaEvent_t, int>> prof_marks; // (event, stage id or -1 for "begin")
    double prof_ms[NNP_N_STAGES];
    int64_t prof_n[NNP_N_STAGES];

    // system
    int n, n_mols, periodic, have_system, have_lists, have_forces, md_ready;
    float box[3];
    // Cells narrower than 2 (rcr + skin) are evaluated as the smallest supercell wide enough for the minimum image: the
    // caller's n_user atoms are copies 0 of n = n_user * rep internal atoms (internal "original" index e = copy * n_user +
    // atom); every output is taken from copy 0 and extensive sums are divided by rep (all periodic images, exactly).
    int n_user, rep, rep_m[3], tric;
    float cell[9];                  // internal (super)cell, rows = lattice vectors; zero: non-periodic
    float cell_user[9];
    int bucket_off[NNP_MAX_SPECIES + 1]; // species-major internal order: atoms of species s are [off[s], off[s+1])
    GridInfo grid;
    float skin, dt;
    // Langevin BAOAB (nnp_md_set_langevin); gamma = 0: velocity Verlet
    float lgv_gamma, lgv_kT, lgv_c1;
    uint64_t lgv_seed;
    float *d_lgv_c2;                // [S] sqrt((1 - c1^2) kT accel_conv / m_s)
    double *d_virial;               // [6] xx yy zz xy xz yz (nnp_energy_forces_virial)
    int want_virial;

    // per-atom state, internal order
    float4 *pos, *pos_tmp; // xyz, w unused
    float4 *vel, *vel_tmp;
    float4 *frc;           // forces (fp32 atomics)
    float4 *rep_stage;     // [3][n_user] replicated small cells in MD: state of copy 0 in caller order (allocated at need)
    int rep_stage_cap;
    float4 *xref;          // positions at the last list build
    int *spc, *spc_tmp;    // species
    int *orig, *orig_tmp;  // internal -> original index
    int *mol, *mol_tmp;    // structure id
    int *mol_offsets;      // [n_mols+1] device copy
    // sort scratch
    int *key, *order, *cell_start, *cursor; // cell_start/cursor: [S*ncell+1]
    int nkeys_cap;
    // lists
    int *nbr_r, *nbr_a;      // [n][cap]
    uint16_t *seg_r, *seg_a; // [n][8] species-segment start offsets; entries S..7 = row length (S <= 7)
    // features and network
    float *G, *dG;           // [n][kpad]
    float *H[3];             // activations / deltas [n_nets][max_atoms][hmax[l]] (one set per network of an ensemble)
    float *e_atom;           // [n]
    double *e_mol;           // [max_mols]
    double *ekin;            // scalar
    int *flags;              // [0] error flags, [1] rebuild request, [2] rebuild count, [4] Langevin step counter
    int *aev_sched;          // [2][NNP_AEV_SCHED_LEN] centre queues of the two AEV kernels (aev.cu), zero between launches
    // staging for the host entry points
    float *io_xyz, *io_vel;  // [n][3]
    double *d_res, *h_res;   // nnp_md_step_host: (epot, ekin, flags[0..2]) packed on the device, read back in one pinned copy
    int *io_species;
    // one MD step as a CUDA graph: kick+drift -> IF(rebuild requested){stage 1} -> stages 2-4 -> kick (nnp_api.cu)
    cudaGraph_t md_graph;
    cudaGraphExec_t md_exec;
    cudaStream_t aux_stream;     // capture stream of the conditional body
    int64_t md_graph_launches;   // kernels per graph launch outside the conditional body
    int no_graph;                // NNP_NO_GRAPH=1: enqueue every step kernel by kernel
    nnp_fused *fused;            // fused MLP chain (mm_mode 4), set up per loaded system
    int no_fused;                // NNP_NO_FUSED=1: always the six-launch path
};

// ---- launches implemented across the .cu files --------------------------------------------------
// neighbor.cu
int nnp_launch_build(nnp_ctx *c, const int *cond_flag); // sort + lists; cond_flag != nullptr: only if *cond_flag != 0
// aev.cu
void nnp_launch_aev_forward(nnp_ctx *c);
void nnp_launch_aev_backward(nnp_ctx *c, float inv_nets, double *d_virial /* [6] or nullptr */);
void nnp_aev_tri_table(uint16_t *h_tri /* [NNP_TRI_LEN] */);
// mlp_simt.cu / mlp_tc.cu
void nnp_launch_gemm_simt(nnp_ctx *c, const GemmBatch &b, int epi, int fp64_acc);
int nnp_launch_gemm_tc(nnp_ctx *c, const GemmBatch &b, int epi, int split3);
// mlp_fused.cu
int nnp_fused_setup(nnp_ctx *c);          // after the layout of a loaded system is known (nnp_set_system)
int nnp_fused_kind(const nnp_ctx *c);     // 0: six launches, 1: whole chain fused, 2: the four middle GEMMs fused
void nnp_launch_mlp_fused(nnp_ctx *c);
void nnp_fused_destroy(nnp_ctx *c);
// integrate.cu
void nnp_launch_kick_drift(nnp_ctx *c);
int nnp_launch_sync_copies(nnp_ctx *c, int what); // replicated small cell: copies := copy 0 (what 0: x + shift and v, 1: F)
void nnp_launch_kick_ke(nnp_ctx *c, int count_step); // count_step: also advance the Langevin step counter flags[4]
void nnp_launch_energy_reduce(nnp_ctx *c);
void nnp_launch_unpermute3(nnp_ctx *c, const float4 *src, float *dst);
void nnp_launch_unpermute3x2(nnp_ctx *c, const float4 *srcA, float *dstA, const float4 *srcB, float *dstB); // both arrays, one launch
void nnp_launch_permute_in3x2(nnp_ctx *c, const float *srcA, float4 *dstA, const float *srcB, float4 *dstB);
void nnp_launch_pack_result(nnp_ctx *c); // d_res = (e_mol[0], ekin, flags[0], flags[1], flags[2])
void nnp_launch_permute_in3(nnp_ctx *c, const float *src, float4 *dst); // dst[i] = src[orig[i]]

void nnp_prof_mark(nnp_ctx *c, int stage); // nnp_api.cu

static inline int nnp_div_up(int a, int b) { return (a + b - 1) / b; }
