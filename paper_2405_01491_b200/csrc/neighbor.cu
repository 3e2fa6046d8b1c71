// Stage 1: O(N) cell-list neighbour build (PAPER.md L41-55 GraphGenerator/GraphFilter, L49 "future releases
// will use cell lists", L341 Verlet skin).  Atoms are re-sorted species-major, cell-minor, so that
//   * every species bucket is one contiguous row range for the grouped MLP GEMMs (stage 3), and
//   * every neighbour row, filled species by species, is automatically grouped by neighbour species
//     (stage 2 needs that: its angular accumulators are per species pair).
// List membership is the fp32 predicate of reading A3: fixed order, round-to-nearest, no FMA.
#include <stdlib.h>

#include "nnp_internal.cuh"

namespace {

constexpr int kWarpsPerBlock = 8;

__device__ __forceinline__ int cell_coord(float x, float L, float invL, float scale, int nc)
{
    float w = x - L * floorf(x * invL); // wrap into [0, L]; rounding can give exactly L
    int c = (int)(w * scale);
    return min(max(c, 0), nc - 1);
}

// cell index and fractional position inside the cell (clamped to [0, 1])
__device__ __forceinline__ int cell_coord_frac(float x, float L, float invL, float scale, int nc, float &f)
{
    const float w = x - L * floorf(x * invL);
    const float cw = w * scale;
    const int c = min(max((int)cw, 0), nc - 1);
    f = fminf(fmaxf(cw - (float)c, 0.f), 1.f);
    return c;
}

// general cell: fractional coordinate c of x, wrapped into [0, 1)
__device__ __forceinline__ float frac_wrapped(const float4 p, const GridInfo &g, int c)
{
    const float s = g.hinv[3 * c] * p.x + g.hinv[3 * c + 1] * p.y + g.hinv[3 * c + 2] * p.z;
    const float w = s - floorf(s);
    return w < 1.0f ? w : 0.0f;
}

__device__ __forceinline__ int cell_of(const float4 p, const GridInfo &g, int mol)
{
    if (!g.periodic) return mol;
    if (g.tric) { // bins cut in fractional coordinates (cell_scale = nc)
        const int cx = min((int)(frac_wrapped(p, g, 0) * g.cell_scale[0]), g.nc[0] - 1);
        const int cy = min((int)(frac_wrapped(p, g, 1) * g.cell_scale[1]), g.nc[1] - 1);
        const int cz = min((int)(frac_wrapped(p, g, 2) * g.cell_scale[2]), g.nc[2] - 1);
        return mol * g.ncell_box + (cz * g.nc[1] + cy) * g.nc[0] + cx;
    }
    int cx = cell_coord(p.x, g.box[0], g.inv_box[0], g.cell_scale[0], g.nc[0]);
    int cy = cell_coord(p.y, g.box[1], g.inv_box[1], g.cell_scale[1], g.nc[1]);
    int cz = cell_coord(p.z, g.box[2], g.inv_box[2], g.cell_scale[2], g.nc[2]);
    return mol * g.ncell_box + (cz * g.nc[1] + cy) * g.nc[0] + cx; // replicas of a periodic batch never share a bin
}

__global__ void k_keys_hist(int n, const float4 *__restrict__ pos, const int *__restrict__ spc,
                            const int *__restrict__ mol, GridInfo g, int *__restrict__ key,
                            int *__restrict__ hist, const int *cond)
{
    if (cond && *cond == 0) return;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int k = spc[i] * g.ncell + cell_of(pos[i], g, mol[i]);
    key[i] = k;
    atomicAdd(&hist[k], 1);
}

// Single-block exclusive scan of hist[0..nk) into start[0..nk]; also clears hist for reuse as cursor.
// A pass covers kScanTiles tiles of 1024 keys (thread t owns key tile * 1024 + t, coalesced): all loads of a pass are
// issued before the first use (one global-memory latency per pass, not one per tile), each tile is scanned inside its
// warps with shuffles, and three block barriers per PASS (warp totals -> per-tile offsets -> tile bases) replace the two
// per tile of a tile-serial scan.  The 98k water box (7 x 17^3 = 34,391 keys) is one pass.
constexpr int kScanTiles = 40;
__global__ void __launch_bounds__(1024) k_scan(int nk, int *__restrict__ hist, int *__restrict__ start, const int *cond)
{
    if (cond && *cond == 0) return;
    __shared__ int ws[kScanTiles][33];   // [tile][warp]: warp totals, then exclusive offsets of the warps inside the tile
    __shared__ int tile_tot[2 * 32];     // tile totals, then exclusive tile bases (carry included)
    __shared__ int carry_s;
    const unsigned kFull = 0xffffffffu;
    const int tid = (int)threadIdx.x, lane = tid & 31, wid = tid >> 5;
    static_assert(kScanTiles <= 64, "tile totals are scanned by one warp, two per lane");
    if (tid == 0) carry_s = 0;
    for (int base = 0; base < nk; base += kScanTiles * 1024) {
        int x[kScanTiles]; // own value, then exclusive prefix inside the warp
#pragma unroll
        for (int k = 0; k < kScanTiles; ++k) {
            const int i = base + k * 1024 + tid;
            x[k] = i < nk ? hist[i] : 0;
        }
#pragma unroll
        for (int k = 0; k < kScanTiles; ++k) {
            if (base + k * 1024 >= nk) { // block-uniform: a tile past the end counts as zeros
                if (lane == 31) ws[k][wid] = 0;
                continue;
            }
            const int i = base + k * 1024 + tid;
            if (i < nk) hist[i] = 0;
            const int v = x[k];
            int sc = v;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int y = __shfl_up_sync(kFull, sc, o);
                if (lane >= o) sc += y;
            }
            if (lane == 31) ws[k][wid] = sc;
            x[k] = sc - v;
        }
        __syncthreads(); // also orders the carry_s of the previous pass / the initial zero
        for (int k = wid; k < kScanTiles; k += 32) { // warp w: offsets of the 32 warps inside tiles w, w + 32
            const int v = ws[k][lane];
            int sc = v;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int y = __shfl_up_sync(kFull, sc, o);
                if (lane >= o) sc += y;
            }
            ws[k][lane] = sc - v;
            if (lane == 31) tile_tot[k] = sc;
        }
        __syncthreads();
        if (wid == 0) { // tile bases
            const int v0 = lane < kScanTiles ? tile_tot[lane] : 0, v1 = lane + 32 < kScanTiles ? tile_tot[lane + 32] : 0;
            int s0 = v0, s1 = v1;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int y0 = __shfl_up_sync(kFull, s0, o), y1 = __shfl_up_sync(kFull, s1, o);
                if (lane >= o) { s0 += y0; s1 += y1; }
            }
            const int carry = carry_s, tot0 = __shfl_sync(kFull, s0, 31), tot1 = __shfl_sync(kFull, s1, 31);
            tile_tot[lane] = carry + s0 - v0;
            tile_tot[lane + 32] = carry + tot0 + s1 - v1;
            if (lane == 0) carry_s = carry + tot0 + tot1;
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < kScanTiles; ++k) {
            const int i = base + k * 1024 + tid;
            if (i < nk) start[i] = tile_tot[k] + ws[k][wid] + x[k];
        }
        __syncthreads(); // ws / tile_tot are rewritten by the next pass
    }
    if (tid == 0) start[nk] = carry_s;
}

__global__ void k_scatter(int n, const int *__restrict__ key, const int *__restrict__ start,
                          int *__restrict__ cursor, int *__restrict__ order, const int *cond)
{
    if (cond && *cond == 0) return;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int k = key[i];
    order[start[k] + atomicAdd(&cursor[k], 1)] = i;
}

// Deterministic order inside each (species, cell) bucket (the scatter's atomics place atoms in arrival order): by previous
// index.  One warp per bucket: lane l holds element l and counts the smaller ones (the indices are distinct) - its rank is
// its place.  (One thread per bucket with an insertion sort in global memory took 30 us at 98k atoms: every shifted element
// was a store followed by a dependent load of the same line from L2.)  Buckets of more than 32 atoms: serial, by lane 0.
__global__ void k_sort_buckets(int nk, const int *__restrict__ start, int *__restrict__ order,
                               int *__restrict__ cursor, const int *cond)
{
    if (cond && *cond == 0) return;
    const unsigned kFull = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const int nwarps = (int)(gridDim.x * blockDim.x) >> 5;
    for (int k = (int)(blockIdx.x * blockDim.x + threadIdx.x) >> 5; k < nk; k += nwarps) {
        if (lane == 0) cursor[k] = 0; // leave the histogram / cursor array zeroed for the next build
        const int a = start[k], len = start[k + 1] - a;
        if (len <= 1) continue;
        if (len <= 32) {
            const int v = lane < len ? order[a + lane] : 0x7fffffff;
            int rank = 0;
            for (int q = 0; q < len; ++q) rank += __shfl_sync(kFull, v, q) < v ? 1 : 0;
            if (lane < len) order[a + rank] = v;
        } else if (lane == 0) {
            const int b = a + len;
            for (int i = a + 1; i < b; ++i) {
                int v = order[i], j = i - 1;
                while (j >= a && order[j] > v) { order[j + 1] = order[j]; --j; }
                order[j + 1] = v;
            }
        }
        __syncwarp();
    }
}

__global__ void k_gather(int n, const int *__restrict__ order, const float4 *__restrict__ pos,
                         const float4 *__restrict__ vel, const int *__restrict__ spc, const int *__restrict__ orig,
                         const int *__restrict__ mol, float4 *__restrict__ pos_o, float4 *__restrict__ vel_o,
                         int *__restrict__ spc_o, int *__restrict__ orig_o, int *__restrict__ mol_o, const int *cond)
{
    if (cond && *cond == 0) return;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int s = order[i];
    pos_o[i] = pos[s];
    vel_o[i] = vel[s];
    spc_o[i] = spc[s];
    orig_o[i] = orig[s];
    mol_o[i] = mol[s];
}

__global__ void k_copyback(int n, const float4 *__restrict__ pos_t, const float4 *__restrict__ vel_t,
                           const int *__restrict__ spc_t, const int *__restrict__ orig_t, const int *__restrict__ mol_t,
                           float4 *__restrict__ pos, float4 *__restrict__ vel, float4 *__restrict__ xref,
                           int *__restrict__ spc, int *__restrict__ orig, int *__restrict__ mol, const int *cond)
{
    if (cond && *cond == 0) return;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float4 p = pos_t[i];
    pos[i] = p;
    xref[i] = p;
    vel[i] = vel_t[i];
    spc[i] = spc_t[i];
    orig[i] = orig_t[i];
    mol[i] = mol_t[i];
}

// Reading A3: dx = xj - xi; dx -= L*rint(dx*invL); r2 = (dx*dx + dy*dy) + dz*dz; every op round-to-nearest,
// never contracted into an FMA.
__device__ __forceinline__ float r2_defined(const float4 a, const float4 b, const GridInfo &g)
{
    float dx = __fsub_rn(b.x, a.x), dy = __fsub_rn(b.y, a.y), dz = __fsub_rn(b.z, a.z);
    if (g.tric) {
        // General cell: the lattice vector k_0 a + k_1 b + k_2 c nearest in fractional coordinates is taken
        // off; exact minimum image for every |d| below half the smallest perpendicular width, which setup_grid enforces.
        const float k0 = rintf(g.hinv[0] * dx + g.hinv[1] * dy + g.hinv[2] * dz);
        const float k1 = rintf(g.hinv[3] * dx + g.hinv[4] * dy + g.hinv[5] * dz);
        const float k2 = rintf(g.hinv[6] * dx + g.hinv[7] * dy + g.hinv[8] * dz);
        dx -= k0 * g.h[0] + k1 * g.h[3] + k2 * g.h[6];
        dy -= k0 * g.h[1] + k1 * g.h[4] + k2 * g.h[7];
        dz -= k0 * g.h[2] + k1 * g.h[5] + k2 * g.h[8];
    } else if (g.periodic) {
        // rint as (x + 1.5 * 2^23) - 1.5 * 2^23: the same value as rintf for |x| < 2^22 (round to nearest even on the integer
        // grid of [2^23, 2^24)), two adds on the FMA pipe instead of an FRND on the quarter-rate XU pipe, which this kernel
        // (three of them and five POPC per 32 candidates) kept 62 % busy
        const float M = 12582912.0f;
        dx = __fsub_rn(dx, __fmul_rn(g.box[0], __fsub_rn(__fadd_rn(__fmul_rn(dx, g.inv_box[0]), M), M)));
        dy = __fsub_rn(dy, __fmul_rn(g.box[1], __fsub_rn(__fadd_rn(__fmul_rn(dy, g.inv_box[1]), M), M)));
        dz = __fsub_rn(dz, __fmul_rn(g.box[2], __fsub_rn(__fadd_rn(__fmul_rn(dz, g.inv_box[2]), M), M)));
    }
    return __fadd_rn(__fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy)), __fmul_rn(dz, dz));
}

// (the orthorhombic branch alone: the one-block-per-cell kernel never sees another cell type)
__device__ __forceinline__ float r2_ortho(const float4 a, const float4 b, const GridInfo &g)
{
    float dx = __fsub_rn(b.x, a.x), dy = __fsub_rn(b.y, a.y), dz = __fsub_rn(b.z, a.z);
    const float M = 12582912.0f;
    dx = __fsub_rn(dx, __fmul_rn(g.box[0], __fsub_rn(__fadd_rn(__fmul_rn(dx, g.inv_box[0]), M), M)));
    dy = __fsub_rn(dy, __fmul_rn(g.box[1], __fsub_rn(__fadd_rn(__fmul_rn(dy, g.inv_box[1]), M), M)));
    dz = __fsub_rn(dz, __fmul_rn(g.box[2], __fsub_rn(__fadd_rn(__fmul_rn(dz, g.inv_box[2]), M), M)));
    return __fadd_rn(__fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy)), __fmul_rn(dz, dz));
}

// One warp per atom.  Per species (rows must stay grouped by neighbour species, stage 2), the candidate cells
// are <= 18 contiguous index ranges of the sorted order: the 3 x 3 (y,z) rows of the stencil, each one or two
// x-ranges (x-adjacent cells are adjacent in the sort).  Lane r fetches the bounds of range r (one load round per
// species instead of a dependent chain per row), a warp scan turns the lengths into one flat candidate list, and
// the lanes walk that list 32 candidates at a time (coalesced float4 loads, ballot compaction into the two rows),
// so a trip is full even where single ranges hold 10-40 atoms.  The non-empty ranges are compacted to the low lanes
// (through shared memory); per trip one REDUX.OR builds the bit mask of the range ends that fall into the trip, and a
// lane's range is (ends before the trip) + popc(mask up to its own bit): no search loop.
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
k_build_lists(int n, int S, unsigned present, const float4 *__restrict__ pos, const int *__restrict__ mol,
              const int *__restrict__ cell_start, GridInfo g, float rl2_r, float rl2_a, float rlm2, int cap_r, int cap_a,
              int *__restrict__ nbr_r, int *__restrict__ nbr_a, uint16_t *__restrict__ seg_r,
              uint16_t *__restrict__ seg_a, int *__restrict__ flags, const int *cond)
{
    if (cond && *cond == 0) return;
    __shared__ int2 cr[kWarpsPerBlock][32]; // compacted non-empty ranges: (inclusive end in the flat list, index offset)
    const unsigned kFull = 0xffffffffu;
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int i = blockIdx.x * kWarpsPerBlock + wib;
    if (i >= n) return;
    const float4 pi = pos[i];
    // range `lane` of the stencil: first / last cell (inside one species block) and whether it exists
    int c_first = 0, c_last = 0, nranges = 1;
    bool rng_ok = true; // false: no atom of this range can be inside the list radius
    if (g.tric) { // general cell: the whole 3 x 3 x 3 stencil of fractional bins (every bin is at least the list radius wide)
        const int cx = min((int)(frac_wrapped(pi, g, 0) * g.cell_scale[0]), g.nc[0] - 1);
        const int cy = min((int)(frac_wrapped(pi, g, 1) * g.cell_scale[1]), g.nc[1] - 1);
        const int cz = min((int)(frac_wrapped(pi, g, 2) * g.cell_scale[2]), g.nc[2] - 1);
        const int nys = g.nc[1] >= 3 ? 3 : g.nc[1], nzs = g.nc[2] >= 3 ? 3 : g.nc[2];
        const int nxs = (g.nc[0] > 3 && (cx == 0 || cx == g.nc[0] - 1)) ? 2 : 1;
        nranges = nzs * nys * nxs;
        const int ix = lane % nxs, t = lane / nxs, iy = t % nys, iz = t / nys;
        const int y = nys == 3 ? (cy + iy + g.nc[1] - 1) % g.nc[1] : iy;
        const int z = nzs == 3 ? (cz + iz + g.nc[2] - 1) % g.nc[2] : iz;
        int xa, xb;
        if (g.nc[0] <= 3) { xa = 0; xb = g.nc[0] - 1; }
        else if (cx == 0) { xa = ix ? g.nc[0] - 1 : 0; xb = ix ? g.nc[0] - 1 : 1; }
        else if (cx == g.nc[0] - 1) { xa = ix ? 0 : cx - 1; xb = ix ? 0 : cx; }
        else { xa = cx - 1; xb = cx + 1; }
        const int rowbase = mol[i] * g.ncell_box + (z * g.nc[1] + y) * g.nc[0];
        c_first = rowbase + xa;
        c_last = rowbase + xb;
    } else if (g.periodic) {
        float fx, fy, fz;
        const int cx = cell_coord_frac(pi.x, g.box[0], g.inv_box[0], g.cell_scale[0], g.nc[0], fx);
        const int cy = cell_coord_frac(pi.y, g.box[1], g.inv_box[1], g.cell_scale[1], g.nc[1], fy);
        const int cz = cell_coord_frac(pi.z, g.box[2], g.inv_box[2], g.cell_scale[2], g.nc[2], fz);
        const int nys = g.nc[1] >= 3 ? 3 : g.nc[1], nzs = g.nc[2] >= 3 ? 3 : g.nc[2]; // distinct cells among c-1, c, c+1
        const int nxs = (g.nc[0] > 3 && (cx == 0 || cx == g.nc[0] - 1)) ? 2 : 1;     // the x range wraps
        nranges = nzs * nys * nxs;
        const int ix = lane % nxs, t = lane / nxs, iy = t % nys, iz = t / nys;
        const int y = nys == 3 ? (cy + iy + g.nc[1] - 1) % g.nc[1] : iy;
        const int z = nzs == 3 ? (cz + iz + g.nc[2] - 1) % g.nc[2] : iz;
        // Trim the stencil with the atom's position inside its cell: a (y,z) row whose nearest point is farther than the
        // list radius (+ 0.01 A for the rounding of the binning) holds no neighbour, and of the three x cells of a row
        // only those within sqrt(rl^2 - d_yz^2) of the atom are needed: ~27 % fewer candidates at cell edge ~ rl.
        // (Only where c-1, c, c+1 are three distinct cells, so that the nearest image lies on the side looked at.)
        float d2 = 0.f;
        if (nys == 3 && iy != 1) { const float dd = (iy == 0 ? fy : 1.0f - fy) * g.box[1] / (float)g.nc[1]; d2 += dd * dd; }
        if (nzs == 3 && iz != 1) { const float dd = (iz == 0 ? fz : 1.0f - fz) * g.box[2] / (float)g.nc[2]; d2 += dd * dd; }
        rng_ok = d2 <= rlm2;
        const float reach2 = rlm2 - d2, lenx = g.box[0] / (float)g.nc[0];
        const bool need_m = (fx * lenx) * (fx * lenx) <= reach2, need_p = ((1.0f - fx) * lenx) * ((1.0f - fx) * lenx) <= reach2;
        int xa, xb;
        if (g.nc[0] <= 3) { xa = 0; xb = g.nc[0] - 1; }
        else if (cx == 0) { xa = ix ? g.nc[0] - 1 : 0; xb = ix ? g.nc[0] - 1 : (need_p ? 1 : 0); if (ix && !need_m) rng_ok = false; }
        else if (cx == g.nc[0] - 1) { xa = ix ? 0 : (need_m ? cx - 1 : cx); xb = ix ? 0 : cx; if (ix && !need_p) rng_ok = false; }
        else { xa = need_m ? cx - 1 : cx; xb = need_p ? cx + 1 : cx; }
        const int rowbase = mol[i] * g.ncell_box + (z * g.nc[1] + y) * g.nc[0];
        c_first = rowbase + xa;
        c_last = rowbase + xb;
    } else {
        c_first = c_last = mol[i]; // the "cell" of a non-periodic structure is the structure itself
    }
    int cnt_r = 0, cnt_a = 0;
    int *row_r = nbr_r + (size_t)i * cap_r;
    int *row_a = nbr_a + (size_t)i * cap_a;
    const unsigned lt = (1u << lane) - 1u;
    int seg_r_l = 0, seg_a_l = 0; // lane s: where the segment of species s starts in the two rows
    for (int s = 0; s < S; ++s) {
        if (lane == s) { seg_r_l = min(cnt_r, cap_r); seg_a_l = min(cnt_a, cap_a); }
        if (!(present >> s & 1u)) continue;
        int beg = 0, len = 0;
        if (lane < nranges && rng_ok) {
            beg = cell_start[s * g.ncell + c_first];
            len = cell_start[s * g.ncell + c_last + 1] - beg;
        }
        int incl = len; // inclusive prefix of the range lengths
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(kFull, incl, o);
            if (lane >= o) incl += y;
        }
        const int total = __shfl_sync(kFull, incl, 31);
        const int off = beg - (incl - len); // flat index v of range r is atom v + off_r
        const unsigned nonempty = __ballot_sync(kFull, len > 0);
        if (len > 0) cr[wib][__popc(nonempty & lt)] = make_int2(incl, off);
        __syncwarp();
        const int2 ce = lane < __popc(nonempty) ? cr[wib][lane] : make_int2(0x7fffffff, 0); // lane k: k-th non-empty range
        __syncwarp();
        int r0 = 0; // non-empty ranges that end before this trip
        for (int t0 = 0; t0 < total; t0 += 32) {
            const int v = t0 + lane;
            const bool act = v < total;
            const unsigned d = (unsigned)(ce.x - t0); // the ends are distinct: one bit per range that ends inside the trip
            const unsigned ends = __reduce_or_sync(kFull, d < 32u ? 1u << d : 0u);
            const int r = r0 + __popc(ends & ((2u << lane) - 1u)); // ranges with end <= v
            r0 += __popc(ends);
            const int j = v + __shfl_sync(kFull, ce.y, r & 31);
            bool hr = false, ha = false;
            if (act && j != i) {
                const float r2 = r2_defined(pi, pos[j], g);
                hr = r2 < rl2_r;
                ha = r2 < rl2_a;
            }
            const unsigned mr = __ballot_sync(kFull, hr);
            const unsigned ma = __ballot_sync(kFull, ha);
            const int p_r = cnt_r + __popc(mr & lt), p_a = cnt_a + __popc(ma & lt);
            if (hr && p_r < cap_r) row_r[p_r] = j;
            if (ha && p_a < cap_a) row_a[p_a] = j;
            cnt_r += __popc(mr);
            cnt_a += __popc(ma);
        }
    }
    if (lane >= S) { seg_r_l = min(cnt_r, cap_r); seg_a_l = min(cnt_a, cap_a); } // entries S..7: the row length
    if (lane < NNP_MAX_SPECIES) {
        seg_r[(size_t)i * NNP_MAX_SPECIES + lane] = (uint16_t)seg_r_l;
        seg_a[(size_t)i * NNP_MAX_SPECIES + lane] = (uint16_t)seg_a_l;
    }
    if (lane == 0) {
        if (cnt_r > cap_r) atomicOr(&flags[0], NNP_FLAG_CAP_R);
        if (cnt_a > cap_a) atomicOr(&flags[0], NNP_FLAG_CAP_A);
    }
}

// The same lists, one block per cell (orthorhombic periodic boxes with at least three cells per dimension): the atoms of the
// 27 stencil cells are staged ONCE in shared memory for all centres of the cell (SURVEY section 6 / north_star: "shared-
// memory staging of neighbour tiles"), wrapped into the box and shifted by the periodic image under which the stencil cell is
// seen from this one, so that a candidate costs a shared-memory load, three subtractions and a sum of squares instead of an
// index-range decode, a global load and a minimum image (~40 against ~78 instructions per 32 candidates; all 27 cells instead
// of the per-atom trimmed stencil: 1.4 times the candidates).  The wrapped and shifted difference is not the arithmetic of
// reading A3, it only agrees with it to rounding: a candidate whose r^2 falls within `band` of a list radius is decided by
// r2_defined() on the two original positions (a few per cent of the centres have one), so the rows are the defined ones.
// band: the staged coordinates and the wrapped centre carry at most ~2 ulp of the largest |coordinate| involved each, so
// |r2' - r2| <= 2 |d|_1 * 4 ulp(M) + rounding of the squares < 32 rl eps M with M = max |x| + 2 L (block maximum).
// A pair whose cell-derived image differs from rint((xj - xi) / L) is at least 1.05 cell widths apart under both: rejected by both.
constexpr int kTileWarps = 4;
constexpr int kTileCap = 1024;   // candidates staged at a time (16 KiB); longer species segments come in windows
constexpr int kTileCen = 128;    // centres of a cell handled at a time
__global__ void __launch_bounds__(kTileWarps * 32)
k_build_lists_tile(int n, int S, unsigned present, const float4 *__restrict__ pos, const int *__restrict__ cell_start, GridInfo g,
                   float rl_r, float rl2_r, float rl2_a, int cap_r, int cap_a, int *__restrict__ nbr_r, int *__restrict__ nbr_a,
                   uint16_t *__restrict__ seg_r, uint16_t *__restrict__ seg_a, int *__restrict__ flags, const int *cond)
{
    if (cond && *cond == 0) return;
    __shared__ float4 cand[kTileCap + 32];            // wrapped + shifted position, w = index as bits (+ padding of the last trip)
    __shared__ int s_rbeg[27], s_pref[28];            // stencil ranges of the current species: first atom, prefix of the lengths
    __shared__ float s_sh[27][3];                     // their image shifts
    __shared__ int s_cen[kTileCen], s_cnt_r[kTileCen], s_cnt_a[kTileCen];
    __shared__ int s_cpref[NNP_MAX_SPECIES + 1];      // centres of the cell per species (prefix)
    __shared__ unsigned s_mmax;
    const unsigned kFull = 0xffffffffu;
    const int tid = threadIdx.x, lane = tid & 31, wib = tid >> 5;
    const int c = blockIdx.x, mol = c / g.ncell_box, cb = c - mol * g.ncell_box;
    const int cx = cb % g.nc[0], cy = (cb / g.nc[0]) % g.nc[1], cz = cb / (g.nc[0] * g.nc[1]);
    if (tid == 0) {
        int acc = 0;
        for (int s = 0; s < S; ++s) { s_cpref[s] = acc; acc += cell_start[s * g.ncell + c + 1] - cell_start[s * g.ncell + c]; }
        for (int s = S; s <= NNP_MAX_SPECIES; ++s) s_cpref[s] = acc;
        s_mmax = 0u;
    }
    __syncthreads();
    const int ncen_all = s_cpref[S];
    if (ncen_all == 0) return;
    auto wrap = [&](float x, int d) { return x - g.box[d] * floorf(x * g.inv_box[d]); }; // as cell_coord(): may give exactly L
    const unsigned lt = (1u << lane) - 1u;
    // (an opaque copy of the staged array's address: the compiler re-derived it from the shared window in every trip)
    uint32_t cand_a = (uint32_t)__cvta_generic_to_shared(cand);
    asm volatile("mov.b32 %0, %0;" : "+r"(cand_a));
    const float4 *cand_w = reinterpret_cast<const float4 *>(__cvta_shared_to_generic(cand_a));
    for (int cen0 = 0; cen0 < ncen_all; cen0 += kTileCen) {
        const int ncen = min(kTileCen, ncen_all - cen0);
        for (int q = tid; q < ncen; q += kTileWarps * 32) {
            const int f = cen0 + q; // f-th centre of the cell: species block s, atom cell_start[s][c] + (f - prefix)
            int s = 0;
            while (f >= s_cpref[s + 1]) ++s;
            s_cen[q] = cell_start[s * g.ncell + c] + (f - s_cpref[s]);
            s_cnt_r[q] = 0;
            s_cnt_a[q] = 0;
        }
        __syncthreads();
        for (int s = 0; s < S; ++s) {
            for (int q = tid; q < ncen; q += kTileWarps * 32) { // where the segment of species s starts in the two rows
                seg_r[(size_t)s_cen[q] * NNP_MAX_SPECIES + s] = (uint16_t)min(s_cnt_r[q], cap_r);
                seg_a[(size_t)s_cen[q] * NNP_MAX_SPECIES + s] = (uint16_t)min(s_cnt_a[q], cap_a);
            }
            if (!(present >> s & 1u)) continue;
            if (wib == 0) { // the 27 stencil cells of this cell for species s
                int len = 0;
                if (lane < 27) {
                    const int dx = lane % 3 - 1, dy = (lane / 3) % 3 - 1, dz = lane / 9 - 1;
                    int x = cx + dx, y = cy + dy, z = cz + dz;
                    float sx = 0.f, sy = 0.f, sz = 0.f;
                    if (x < 0) { x += g.nc[0]; sx = -g.box[0]; } else if (x >= g.nc[0]) { x -= g.nc[0]; sx = g.box[0]; }
                    if (y < 0) { y += g.nc[1]; sy = -g.box[1]; } else if (y >= g.nc[1]) { y -= g.nc[1]; sy = g.box[1]; }
                    if (z < 0) { z += g.nc[2]; sz = -g.box[2]; } else if (z >= g.nc[2]) { z -= g.nc[2]; sz = g.box[2]; }
                    const int cc = s * g.ncell + mol * g.ncell_box + (z * g.nc[1] + y) * g.nc[0] + x;
                    const int beg = cell_start[cc];
                    len = cell_start[cc + 1] - beg;
                    s_rbeg[lane] = beg;
                    s_sh[lane][0] = sx; s_sh[lane][1] = sy; s_sh[lane][2] = sz;
                }
                int incl = len;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int y = __shfl_up_sync(kFull, incl, o);
                    if (lane >= o) incl += y;
                }
                if (lane < 27) s_pref[lane + 1] = incl;
                if (lane == 0) s_pref[0] = 0;
            }
            __syncthreads();
            const int total = s_pref[27];
            for (int w0 = 0; w0 < total; w0 += kTileCap) {
                const int nw = min(kTileCap, total - w0);
                float mloc = 0.f;
                for (int v = tid; v < nw; v += kTileWarps * 32) {
                    const int flat = w0 + v;
                    int r = 0; // range of the flat index: s_pref[r] <= flat < s_pref[r + 1] (27 entries: five halvings)
#pragma unroll
                    for (int st = 16; st >= 1; st >>= 1)
                        if (r + st <= 26 && s_pref[r + st] <= flat) r += st;
                    const int j = s_rbeg[r] + (flat - s_pref[r]);
                    const float4 p = pos[j];
                    mloc = fmaxf(mloc, fmaxf(fabsf(p.x), fmaxf(fabsf(p.y), fabsf(p.z))));
                    cand[v] = make_float4(wrap(p.x, 0) + s_sh[r][0], wrap(p.y, 1) + s_sh[r][1], wrap(p.z, 2) + s_sh[r][2], __int_as_float(j));
                }
                for (int v = nw + tid; v < ((nw + 31) & ~31); v += kTileWarps * 32) // pad the last trip: never a neighbour
                    cand[v] = make_float4(3.0e18f, 3.0e18f, 3.0e18f, __int_as_float(-1));
                const unsigned mw = __reduce_max_sync(kFull, __float_as_uint(mloc)); // (non-negative floats order as integers)
                if (lane == 0) atomicMax(&s_mmax, mw);
                __syncthreads();
                for (int q = wib; q < ncen; q += kTileWarps) {
                    const int i = s_cen[q];
                    const float4 pi = pos[i];
                    const float mi = fmaxf(fabsf(pi.x), fmaxf(fabsf(pi.y), fabsf(pi.z)));
                    const float M = fmaxf(__uint_as_float(s_mmax), mi) + 2.0f * fmaxf(g.box[0], fmaxf(g.box[1], g.box[2]));
                    const float band = 32.0f * rl_r * 1.1920929e-7f * M;
                    const float wx = wrap(pi.x, 0), wy = wrap(pi.y, 1), wz = wrap(pi.z, 2);
                    const int cnt_r0 = s_cnt_r[q], cnt_a0 = s_cnt_a[q];
                    // this lane's next free slot in the two rows (a pointer that moves with the row, no index arithmetic per
                    // store) and the slots left; rows that are full count on but store nothing
                    int *dst_r = nbr_r + (size_t)i * cap_r + cnt_r0, *dst_a = nbr_a + (size_t)i * cap_a + cnt_a0;
                    int left_r = cap_r - cnt_r0, left_a = cap_a - cnt_a0, cnt_r = cnt_r0, cnt_a = cnt_a0;
                    const float4 *cv = cand_w + lane;
                    const int ntrip = (nw + 31) >> 5;
                    for (int t = 0; t < ntrip; ++t, cv += 32) {
                        const float4 cj = *cv;
                        const int j = __float_as_int(cj.w);
                        const float dx = cj.x - wx, dy = cj.y - wy, dz = cj.z - wz;
                        float r2 = dx * dx + dy * dy + dz * dz;
                        if ((fabsf(r2 - rl2_r) <= band || fabsf(r2 - rl2_a) <= band) && j >= 0) r2 = r2_ortho(pi, pos[j], g);
                        const bool hr = r2 < rl2_r && j != i, ha = r2 < rl2_a && j != i;
                        const unsigned mr = __ballot_sync(kFull, hr);
                        const unsigned ma = __ballot_sync(kFull, ha);
                        const int o_r = __popc(mr & lt), o_a = __popc(ma & lt), n_r = __popc(mr), n_a = __popc(ma);
                        if (hr && o_r < left_r) dst_r[o_r] = j;
                        if (ha && o_a < left_a) dst_a[o_a] = j;
                        dst_r += n_r; dst_a += n_a;
                        left_r -= n_r; left_a -= n_a;
                        cnt_r += n_r; cnt_a += n_a;
                    }
                    if (lane == 0) { s_cnt_r[q] = cnt_r; s_cnt_a[q] = cnt_a; }
                }
                __syncthreads();
            }
            __syncthreads(); // (a species without candidates: nobody reads the range table any more before it is rewritten)
        }
        for (int q = tid; q < ncen; q += kTileWarps * 32) { // entries S..7: the row length
            const int i = s_cen[q], cr_ = s_cnt_r[q], ca_ = s_cnt_a[q];
            for (int s = S; s < NNP_MAX_SPECIES; ++s) {
                seg_r[(size_t)i * NNP_MAX_SPECIES + s] = (uint16_t)min(cr_, cap_r);
                seg_a[(size_t)i * NNP_MAX_SPECIES + s] = (uint16_t)min(ca_, cap_a);
            }
            if (cr_ > cap_r) atomicOr(&flags[0], NNP_FLAG_CAP_R);
            if (ca_ > cap_a) atomicOr(&flags[0], NNP_FLAG_CAP_A);
        }
        __syncthreads();
    }
}

__global__ void k_finish_build(int *flags, const int *cond)
{
    if (cond && *cond == 0) return;
    flags[1] = 0;
    flags[2] += 1;
}

} // namespace

int nnp_launch_build(nnp_ctx *c, const int *cond)
{
    const int n = c->n, S = c->S;
    const int nk = S * c->grid.ncell;
    const int T = 256, nb = nnp_div_up(n, T);
    cudaStream_t st = c->stream;
    // c->cursor doubles as the histogram; it is zero on entry (cleared at create and by k_sort_buckets)
    k_keys_hist<<<nb, T, 0, st>>>(n, c->pos, c->spc, c->mol, c->grid, c->key, c->cursor, cond);
    k_scan<<<1, 1024, 0, st>>>(nk, c->cursor, c->cell_start, cond);
    k_scatter<<<nb, T, 0, st>>>(n, c->key, c->cell_start, c->cursor, c->order, cond);
    {
        const int want = nnp_div_up(nk, T / 32), cap = 148 * 8;
        k_sort_buckets<<<want < cap ? want : cap, T, 0, st>>>(nk, c->cell_start, c->order, c->cursor, cond);
    }
    k_gather<<<nb, T, 0, st>>>(n, c->order, c->pos, c->vel, c->spc, c->orig, c->mol, c->pos_tmp, c->vel_tmp,
                               c->spc_tmp, c->orig_tmp, c->mol_tmp, cond);
    k_copyback<<<nb, T, 0, st>>>(n, c->pos_tmp, c->vel_tmp, c->spc_tmp, c->orig_tmp, c->mol_tmp, c->pos, c->vel,
                                 c->xref, c->spc, c->orig, c->mol, cond);
    const float rl_r = c->aev.rcr + c->skin, rl_a = c->aev.rca + c->skin;
    // one block per cell where every dimension has three distinct stencil cells (NNP_LIST_TILE=0: the warp-per-atom kernel)
    const char *tile_env = getenv("NNP_LIST_TILE"); // (read per build: a test switches it)
    const bool tile_on = !(tile_env && atoi(tile_env) == 0);
    if (tile_on && c->grid.periodic && !c->grid.tric && c->grid.nc[0] >= 3 && c->grid.nc[1] >= 3 && c->grid.nc[2] >= 3)
        k_build_lists_tile<<<c->grid.ncell, kTileWarps * 32, 0, st>>>(n, S, c->present_mask, c->pos, c->cell_start, c->grid, rl_r, rl_r * rl_r,
                                                                      rl_a * rl_a, c->aev.cap_r, c->aev.cap_a, c->nbr_r, c->nbr_a, c->seg_r,
                                                                      c->seg_a, c->flags, cond);
    else
    k_build_lists<<<nnp_div_up(n, kWarpsPerBlock), kWarpsPerBlock * 32, 0, st>>>(
        n, S, c->present_mask, c->pos, c->mol, c->cell_start, c->grid, rl_r * rl_r, rl_a * rl_a, (rl_r + 0.01f) * (rl_r + 0.01f),
        c->aev.cap_r, c->aev.cap_a,
        c->nbr_r, c->nbr_a, c->seg_r, c->seg_a, c->flags, cond);
    k_finish_build<<<1, 1, 0, st>>>(c->flags, cond);
    if (!cond) c->launches += 8; // conditional builds are counted from the device-side rebuild counter (flags[2])
    return 0;
}
