// nnp_neighbors_no_alloc: fixed-radius neighbour lists of one point set with NO allocation of any kind - for callers that
// cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it).  It is the cell-list
// build of stage 1 (neighbor.cu: keys + histogram, scan, scatter, list kernel; PAPER.md L41-55, L49 cell lists) cut down to one
// species, one structure, one radius and an orthorhombic box, with every piece of its scratch memory - wrapped positions,
// cell keys, the sorted order, the cell histogram / cursor and the cell start table - in ONE file-scope device array of a
// fixed size instead of buffers owned by an nnp_ctx.  List membership is the fp32 predicate of reading A3, the
// same arithmetic in the same order as r2_defined() in neighbor.cu, so the rows equal those of nnp_build_neighbors.
//
// The array is part of the library image: every GPU that loads libnnp_b200.so holds NA_SCRATCH_BYTES (~450 KiB) until the
// process exits.  In host code its NAME is a host-side stand-in, not a device address (a kernel given it would fault, or,
// where the GPU can reach host memory, silently use the wrong memory): the address is asked for once per device, with that
// device current, with cudaGetSymbolAddress() below, and only that pointer is handed to the kernels.
// All calls share the array and it keeps the last call's contents: what must start at zero (the cell histogram) is cleared at
// the start of every call; two calls that overlap on one GPU (different streams, or graph launches that run concurrently)
// RACE on it - serialise them.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "../../include/nnp.h"

namespace {

constexpr int NA_MAX_ATOMS = NNP_NO_ALLOC_MAX_ATOMS; // 16384
constexpr int NA_MAX_CELLS = 8192;                   // 20^3 = 8000 cells of one list radius
constexpr int NA_WARPS = 8;

// layout of the scratch array (offsets in bytes, each a multiple of 256)
constexpr size_t NA_OFF_POS = 0;                                               // float4 [NA_MAX_ATOMS]: positions, w unused
constexpr size_t NA_OFF_KEY = NA_OFF_POS + sizeof(float4) * NA_MAX_ATOMS;      // int [NA_MAX_ATOMS]: cell of atom i
constexpr size_t NA_OFF_ORDER = NA_OFF_KEY + sizeof(int) * NA_MAX_ATOMS;       // int [NA_MAX_ATOMS]: atoms grouped by cell
constexpr size_t NA_OFF_CURSOR = NA_OFF_ORDER + sizeof(int) * NA_MAX_ATOMS;    // int [NA_MAX_CELLS]: histogram, then cursor
constexpr size_t NA_OFF_START = NA_OFF_CURSOR + sizeof(int) * NA_MAX_CELLS;    // int [NA_MAX_CELLS + 1] (+ padding)
constexpr size_t NA_SCRATCH_BYTES = NA_OFF_START + sizeof(int) * NA_MAX_CELLS + 256;
static_assert(NA_OFF_KEY % 256 == 0 && NA_OFF_ORDER % 256 == 0 && NA_OFF_CURSOR % 256 == 0 && NA_OFF_START % 256 == 0, "alignment");

static __device__ __align__(256) unsigned char g_na_scratch[NA_SCRATCH_BYTES];

struct NaGrid {
    int nc[3], ncell, periodic;
    float box[3], inv_box[3], scale[3]; // inv_box = 1.0f / box (IEEE division on the host), scale = nc / box
};

__device__ __forceinline__ int na_cell_coord(float x, float L, float invL, float scale, int nc)
{
    const float w = x - L * floorf(x * invL); // wrap into [0, L]; rounding can give exactly L
    const int c = (int)(w * scale);
    return min(max(c, 0), nc - 1);
}

__device__ __forceinline__ int na_cell_of(const float4 p, const NaGrid &g)
{
    if (!g.periodic) return 0; // a non-periodic point set is one cell
    const int cx = na_cell_coord(p.x, g.box[0], g.inv_box[0], g.scale[0], g.nc[0]);
    const int cy = na_cell_coord(p.y, g.box[1], g.inv_box[1], g.scale[1], g.nc[1]);
    const int cz = na_cell_coord(p.z, g.box[2], g.inv_box[2], g.scale[2], g.nc[2]);
    return (cz * g.nc[1] + cy) * g.nc[0] + cx;
}

// Reading A3, as r2_defined() in neighbor.cu: dx = xj - xi; dx -= L * rint(dx * invL); r2 = (dx dx + dy dy) + dz dz,
// every operation rounded to nearest, none contracted into an FMA.
__device__ __forceinline__ float na_r2(const float4 a, const float4 b, const NaGrid &g)
{
    float dx = __fsub_rn(b.x, a.x), dy = __fsub_rn(b.y, a.y), dz = __fsub_rn(b.z, a.z);
    if (g.periodic) {
        dx = __fsub_rn(dx, __fmul_rn(g.box[0], rintf(__fmul_rn(dx, g.inv_box[0]))));
        dy = __fsub_rn(dy, __fmul_rn(g.box[1], rintf(__fmul_rn(dy, g.inv_box[1]))));
        dz = __fsub_rn(dz, __fmul_rn(g.box[2], rintf(__fmul_rn(dz, g.inv_box[2]))));
    }
    return __fadd_rn(__fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy)), __fmul_rn(dz, dz));
}

// positions -> float4 copy, cell key, cell histogram (hist must be zero on entry)
__global__ void k_na_keys(int n, const float *__restrict__ xyz, NaGrid g, float4 *__restrict__ pos, int *__restrict__ key,
                          int *__restrict__ hist)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float4 p = make_float4(xyz[3 * i], xyz[3 * i + 1], xyz[3 * i + 2], 0.f);
    pos[i] = p;
    const int k = na_cell_of(p, g);
    key[i] = k;
    atomicAdd(&hist[k], 1);
}

// Single-block exclusive scan of hist[0..nk) into start[0..nk]; clears hist for its second life as the scatter cursor.
// Thread t owns the keys [t * per, (t + 1) * per); nk <= NA_MAX_CELLS = 8 per thread.
__global__ void __launch_bounds__(1024) k_na_scan(int nk, int *__restrict__ hist, int *__restrict__ start)
{
    __shared__ int wsum[32];
    const unsigned kFull = 0xffffffffu;
    const int tid = (int)threadIdx.x, lane = tid & 31, wid = tid >> 5;
    constexpr int per = NA_MAX_CELLS / 1024;
    int v[per], tot = 0;
#pragma unroll
    for (int q = 0; q < per; ++q) {
        const int k = tid * per + q;
        v[q] = k < nk ? hist[k] : 0;
        if (k < nk) hist[k] = 0;
        tot += v[q];
    }
    int sc = tot;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int y = __shfl_up_sync(kFull, sc, o);
        if (lane >= o) sc += y;
    }
    if (lane == 31) wsum[wid] = sc;
    __syncthreads();
    if (wid == 0) {
        const int w = wsum[lane];
        int ws = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(kFull, ws, o);
            if (lane >= o) ws += y;
        }
        wsum[lane] = ws - w;
    }
    __syncthreads();
    int run = wsum[wid] + sc - tot; // exclusive prefix of this thread's first key
#pragma unroll
    for (int q = 0; q < per; ++q) {
        const int k = tid * per + q;
        if (k < nk) start[k] = run;
        run += v[q];
    }
    if (tid == 1023) start[nk] = run; // (keys past nk count as zeros: run is the total)
}

__global__ void k_na_scatter(int n, const int *__restrict__ key, const int *__restrict__ start, int *__restrict__ cursor,
                             int *__restrict__ order)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int k = key[i];
    order[start[k] + atomicAdd(&cursor[k], 1)] = i;
}

// One warp per atom: the candidate cells are the distinct cells among c - 1, c, c + 1 per dimension; per (y, z) row of the
// stencil one or two x ranges that are contiguous in `order`.  32 candidates per trip, ballot compaction into the row.
// counts[i] is the number of neighbours found; entries beyond `stride` are not stored (the caller compares).
__global__ void __launch_bounds__(NA_WARPS * 32)
k_na_lists(int n, NaGrid g, float rc2, const float4 *__restrict__ pos, const int *__restrict__ order,
           const int *__restrict__ start, int *__restrict__ counts, int *__restrict__ list, int stride)
{
    const unsigned kFull = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const int i = blockIdx.x * NA_WARPS + (threadIdx.x >> 5);
    if (i >= n) return;
    const float4 pi = pos[i];
    int cx = 0, cy = 0, cz = 0;
    if (g.periodic) {
        cx = na_cell_coord(pi.x, g.box[0], g.inv_box[0], g.scale[0], g.nc[0]);
        cy = na_cell_coord(pi.y, g.box[1], g.inv_box[1], g.scale[1], g.nc[1]);
        cz = na_cell_coord(pi.z, g.box[2], g.inv_box[2], g.scale[2], g.nc[2]);
    }
    const int nys = g.nc[1] >= 3 ? 3 : g.nc[1], nzs = g.nc[2] >= 3 ? 3 : g.nc[2];
    const int nxs = (g.nc[0] > 3 && (cx == 0 || cx == g.nc[0] - 1)) ? 2 : 1; // the x range wraps
    const unsigned lt = (1u << lane) - 1u;
    int cnt = 0;
    int *row = list + (size_t)i * stride;
    for (int iz = 0; iz < nzs; ++iz)
        for (int iy = 0; iy < nys; ++iy)
            for (int ix = 0; ix < nxs; ++ix) {
                const int y = nys == 3 ? (cy + iy + g.nc[1] - 1) % g.nc[1] : iy;
                const int z = nzs == 3 ? (cz + iz + g.nc[2] - 1) % g.nc[2] : iz;
                int xa, xb;
                if (g.nc[0] <= 3) { xa = 0; xb = g.nc[0] - 1; }
                else if (cx == 0) { xa = ix ? g.nc[0] - 1 : 0; xb = ix ? g.nc[0] - 1 : 1; }
                else if (cx == g.nc[0] - 1) { xa = ix ? 0 : cx - 1; xb = ix ? 0 : cx; }
                else { xa = cx - 1; xb = cx + 1; }
                const int rowbase = (z * g.nc[1] + y) * g.nc[0];
                const int beg = start[rowbase + xa], end = start[rowbase + xb + 1];
                for (int v0 = beg; v0 < end; v0 += 32) {
                    const int v = v0 + lane;
                    bool hit = false;
                    int j = -1;
                    if (v < end) {
                        j = order[v];
                        if (j != i) hit = na_r2(pi, pos[j], g) < rc2;
                    }
                    const unsigned m = __ballot_sync(kFull, hit);
                    const int p = cnt + __popc(m & lt);
                    if (hit && p < stride) row[p] = j;
                    cnt += __popc(m);
                }
            }
    if (lane == 0) counts[i] = cnt;
}

thread_local char g_na_err[256] = "";
void *g_na_ptr[64] = {nullptr}; // device address of g_na_scratch per device (filled at the first call on that device)

} // namespace

extern "C" {

const char *nnp_neighbors_no_alloc_error(void) { return g_na_err; }

int nnp_neighbors_no_alloc(int n_atoms, const float *d_xyz, const float h_box[3], float rcut, int32_t *d_counts,
                           int32_t *d_list, int stride, void *cuda_stream)
{
#define NA_FAIL(code, ...) do { snprintf(g_na_err, sizeof(g_na_err), __VA_ARGS__); return (code); } while (0)
#define NA_CU(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) NA_FAIL(NNP_ECUDA, "%s: %s", #x, cudaGetErrorString(e_)); } while (0)
    g_na_err[0] = 0;
    if (n_atoms < 0 || stride < 1 || !(rcut > 0.f)) NA_FAIL(NNP_EINVAL, "nnp_neighbors_no_alloc: n_atoms >= 0, stride >= 1 and rcut > 0 are required");
    if (n_atoms > NA_MAX_ATOMS)
        NA_FAIL(NNP_EINVAL, "nnp_neighbors_no_alloc: %d atoms exceed the fixed scratch of NNP_NO_ALLOC_MAX_ATOMS = %d atoms; use nnp_create / nnp_build_neighbors",
                n_atoms, NA_MAX_ATOMS);
    if (n_atoms == 0) return NNP_OK;
    if (!d_xyz || !d_counts || !d_list) NA_FAIL(NNP_EINVAL, "nnp_neighbors_no_alloc: null argument");

    NaGrid g;
    g.periodic = h_box && (h_box[0] != 0.f || h_box[1] != 0.f || h_box[2] != 0.f);
    for (int d = 0; d < 3; ++d) { g.nc[d] = 1; g.box[d] = 0.f; g.inv_box[d] = 0.f; g.scale[d] = 0.f; }
    if (g.periodic) {
        for (int d = 0; d < 3; ++d) {
            if (!(h_box[d] >= 2.0f * rcut))
                NA_FAIL(NNP_EBOX, "nnp_neighbors_no_alloc: box edge %d = %g is below 2 rcut = %g: the minimum image is not unique", d, h_box[d], 2.0f * rcut);
            g.box[d] = h_box[d];
            g.inv_box[d] = 1.0f / h_box[d];
            int nc = (int)(h_box[d] / (rcut * 1.0001f)); // cells at least one radius wide (+ margin for the rounding of the binning)
            g.nc[d] = nc < 1 ? 1 : nc;
        }
        while ((long long)g.nc[0] * g.nc[1] * g.nc[2] > NA_MAX_CELLS) { // fewer, wider cells: still correct
            const int d = g.nc[0] >= g.nc[1] && g.nc[0] >= g.nc[2] ? 0 : (g.nc[1] >= g.nc[2] ? 1 : 2);
            g.nc[d] -= 1;
        }
        for (int d = 0; d < 3; ++d) g.scale[d] = (float)g.nc[d] / g.box[d];
    }
    g.ncell = g.nc[0] * g.nc[1] * g.nc[2];

    // set-up, once per device and with that device current: the device address of the scratch array
    int dev = -1;
    NA_CU(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) NA_FAIL(NNP_EINVAL, "nnp_neighbors_no_alloc: device index %d is outside the table of 64", dev);
    if (!g_na_ptr[dev]) {
        void *p = nullptr;
        NA_CU(cudaGetSymbolAddress(&p, g_na_scratch));
        if (!p) NA_FAIL(NNP_ECUDA, "nnp_neighbors_no_alloc: cudaGetSymbolAddress returned a null address");
        g_na_ptr[dev] = p;
    }
    unsigned char *base = static_cast<unsigned char *>(g_na_ptr[dev]);
    float4 *pos = reinterpret_cast<float4 *>(base + NA_OFF_POS);
    int *key = reinterpret_cast<int *>(base + NA_OFF_KEY), *order = reinterpret_cast<int *>(base + NA_OFF_ORDER);
    int *cursor = reinterpret_cast<int *>(base + NA_OFF_CURSOR), *start = reinterpret_cast<int *>(base + NA_OFF_START);

    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const int T = 256, nb = (n_atoms + T - 1) / T;
    // the array keeps what the last call left (its cursor holds that call's cell counts): the histogram starts at zero
    NA_CU(cudaMemsetAsync(cursor, 0, sizeof(int) * (size_t)g.ncell, st));
    k_na_keys<<<nb, T, 0, st>>>(n_atoms, d_xyz, g, pos, key, cursor);
    k_na_scan<<<1, 1024, 0, st>>>(g.ncell, cursor, start);
    k_na_scatter<<<nb, T, 0, st>>>(n_atoms, key, start, cursor, order);
    k_na_lists<<<(n_atoms + NA_WARPS - 1) / NA_WARPS, NA_WARPS * 32, 0, st>>>(n_atoms, g, rcut * rcut, pos, order, start, d_counts, d_list, stride);
    NA_CU(cudaGetLastError());
    return NNP_OK;
#undef NA_CU
#undef NA_FAIL
}

} // extern "C"
