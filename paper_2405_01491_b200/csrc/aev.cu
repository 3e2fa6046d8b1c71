// Stage 2 (AEV forward) and the AEV half of stage 4 (reverse pass + force scatter).
// Definition: SURVEY.md 8(c) O2/O3/O6 (PAPER.md L61 cosine switch, L79 Gaussian radial basis, L443 angular form
// (0.5+0.5cos(theta-theta_n))^zeta, L55 pairs of edges with a common centre, L65/L176 forces by reverse mode).
//
// One centre atom per warp at a time (forward: persistent warps, centres handed out by a ticket counter; reverse: two
// consecutive centres per warp of a plain grid - CentreQueue below).  Neighbour rows are grouped by neighbour species (stage 1).  Arithmetic of the inner
// loops is packed f32x2 (FFMA2 / FMUL2 / FADD2, one issue slot for two lanes of math); the forward kernel evaluates
// uniformly spaced shift sets by a Gaussian ladder (AevParams::ladder).
//   loads:   the species-segment table of the NEXT centre is fetched one centre ahead; for the current centre all
//            neighbour indices (radial trips + angular chunks) are loaded first, then all their positions, so one
//            centre costs one index->position latency chain instead of one per loop trip.
//   radial:  the 32 lanes are split among the species segments of the radial row in proportion to their lengths
//            (every lane serves one species, so its 16 Gaussian accumulators belong to one species); the lanes'
//            accumulators are transposed through shared memory and summed per species.
//   angular: the in-cutoff neighbours are compacted into shared memory (dx,dy,dz,r | fc,1/r | fc'), still grouped
//            by species.  The pairs (j,k) of ALL species-pair blocks are processed in one loop: the lanes are split
//            among the non-empty blocks in proportion to their pair counts (one block per lane: its 8x4
//            accumulators belong to one block), which takes ~ceil(pairs/32) trips instead of one ragged loop per
//            block.  Accumulators go through the same shared-memory transpose; lane = feature sums the rows of
//            each block -> one coalesced 128 B store per block.  Triplets are enumerated on the fly and never
//            stored (the paper's GraphAngularExtension stores them, L55).
//   reverse: per pair only three scalars (alpha_j, alpha_k, beta with dE/dd_ij = alpha_j d_ij + beta d_ik) are
//            parked in two per-warp na x na shared-memory matrices; a second pass with lane = neighbour sums its
//            row into the neighbour force without atomics; one 16-byte vector reduction per neighbour goes to
//            global memory.
// cos(theta' - ShfZ) with theta' = acos(0.95 cos theta) is expanded as c' cos ShfZ + sqrt(1-c'^2) sin ShfZ: no acos;
// |c'| <= 0.95 keeps sqrt(1-c'^2) >= 0.31 and (1+cos(theta'-ShfZ))/2 >= 0.1, so neither needs a clamp.
// Columns of G are the active ones of the loaded system (AevParams::cmap / plist, nnp_internal.cuh).
#include "nnp_internal.cuh"

namespace {

#ifndef AEV_FWD_MINB
#define AEV_FWD_MINB 8
#endif
#ifndef AEV_BWD_MINB
#define AEV_BWD_MINB 5
#endif
constexpr int kWarps = 4;
constexpr int kCapA = 64;        // shared-memory slots for in-cutoff angular neighbours per centre
constexpr int kMat = 32;         // reverse pass: pair matrices cover na <= 32 in-cutoff neighbours, beyond: atomics
constexpr int kMatLd = 33;
constexpr int kRedLd = 36;       // row stride of the transpose buffer (conflict-free 16-byte rows / 4-byte columns)
constexpr int KR = 3;            // radial trips whose loads are issued up front (3 x 32 lanes >= typical row)
constexpr int KA = 2;            // angular chunks of 32 loaded up front (cap_a = 64)
constexpr unsigned kFull = 0xffffffffu;
static_assert(kCapA * (kCapA - 1) / 2 == NNP_TRI_LEN, "pair decode table length");

struct WarpSmem {
    float4 d[kCapA];   // dx, dy, dz, r
    float2 fr[kCapA];  // fc, 1/r
    float red[32 * kRedLd];
    int seg[NNP_MAX_SPECIES + 1]; // offsets of the compact-species segments in d[]
    int own[32];
};
struct WarpSmemBwd {
    float4 d[kCapA];
    float2 fr[kCapA];
    float dfc[kCapA];
    int j[kCapA];
    int seg[NNP_MAX_SPECIES + 1];
    int own[32];
    float2 ab[kMat * kMatLd]; // ab[a][b] = (alpha of a in pair (a,b), beta(a,b) = beta(b,a)); fallback path: f[kCapA][3] aliases it
};

__device__ __forceinline__ float ex2(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float lg2(float x)
{
    float y;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rcp(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rsq(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Packed fp32 pairs (FFMA2 / FMUL2 / FADD2 on sm_100): one issue slot for two lanes of arithmetic.  A float2 built as
// (s, s) from one scalar compiles to the scalar-broadcast operand form, no extra moves.
__device__ __forceinline__ float2 fma2(const float2 a, const float2 b, const float2 c)
{
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;"
        : "=l"(d)
        : "l"(*reinterpret_cast<const unsigned long long *>(&a)), "l"(*reinterpret_cast<const unsigned long long *>(&b)),
          "l"(*reinterpret_cast<const unsigned long long *>(&c)));
    return *reinterpret_cast<float2 *>(&d);
}
__device__ __forceinline__ float2 mul2(const float2 a, const float2 b)
{
    unsigned long long d;
    asm("mul.rn.f32x2 %0, %1, %2;"
        : "=l"(d)
        : "l"(*reinterpret_cast<const unsigned long long *>(&a)), "l"(*reinterpret_cast<const unsigned long long *>(&b)));
    return *reinterpret_cast<float2 *>(&d);
}
__device__ __forceinline__ float2 add2(const float2 a, const float2 b)
{
    unsigned long long d;
    asm("add.rn.f32x2 %0, %1, %2;"
        : "=l"(d)
        : "l"(*reinterpret_cast<const unsigned long long *>(&a)), "l"(*reinterpret_cast<const unsigned long long *>(&b)));
    return *reinterpret_cast<float2 *>(&d);
}
__device__ __forceinline__ float2 bc2(const float s) { return make_float2(s, s); }

// TRIC: general cell (a template parameter of the kernels: the orthorhombic kernels carry none of it)
template <bool TRIC>
__device__ __forceinline__ float3 min_image(const float4 a, const float4 b, const AevParams &P)
{
    float dx = b.x - a.x, dy = b.y - a.y, dz = b.z - a.z;
    if (TRIC) { // take off the lattice vector nearest in fractional coordinates (neighbor.cu r2_defined)
        const float M = 12582912.0f;
        const float k0 = (P.hinv[0] * dx + P.hinv[1] * dy + P.hinv[2] * dz + M) - M;
        const float k1 = (P.hinv[3] * dx + P.hinv[4] * dy + P.hinv[5] * dz + M) - M;
        const float k2 = (P.hinv[6] * dx + P.hinv[7] * dy + P.hinv[8] * dz + M) - M;
        dx -= k0 * P.h[0] + k1 * P.h[3] + k2 * P.h[6];
        dy -= k0 * P.h[1] + k1 * P.h[4] + k2 * P.h[7];
        dz -= k0 * P.h[2] + k1 * P.h[5] + k2 * P.h[8];
    } else if (P.periodic) {
        // round-to-nearest by the 1.5 * 2^23 trick: two FADDs on the FMA pipe instead of an FRND on the XU pipe
        // (|d / L| < 2^22 always); any consistent choice of image is fine here, list membership is decided in stage 1
        const float M = 12582912.0f;
        dx -= P.box[0] * ((dx * P.inv_box[0] + M) - M);
        dy -= P.box[1] * ((dy * P.inv_box[1] + M) - M);
        dz -= P.box[2] * ((dz * P.inv_box[2] + M) - M);
    }
    return make_float3(dx, dy, dz);
}

// Species-pair block (compact indices cs <= ct) served by lane b < np(np+1)/2 when it acts as "block lane".
__device__ __forceinline__ void block_of_lane(int np, int lane, int &bcs, int &bct)
{
    bcs = 0; bct = 0;
    if (lane < np * (np + 1) / 2) {
        int off = 0;
        while (lane >= off + (np - bcs)) { off += np - bcs; ++bcs; }
        bct = bcs + (lane - off);
    }
}

// Lane partition: "block lane" b holds a work list of n_b items (0 for lanes that own no block) and a tag.
// Finds the smallest trip count I with sum_b ceil(n_b / I) <= 32 and gives block b the worker lanes
// [beg_b, beg_b + L_b), L_b = ceil(n_b / I).  Worker r of a block takes items r, r + L, r + 2L, ...
struct LanePart {
    int I;          // trips (warp-uniform); 0: nothing to do
    int beg_b, L_b; // as block lane
    int tag;        // as worker: tag of the block served
    int r, L;       // as worker: rank inside the block's lane group and its size; active iff r < L
    unsigned starts; // bit l set: a lane group starts at lane l (warp-uniform)
};
__device__ __forceinline__ LanePart partition(int n_b, int tag_b, int *own, int lane)
{
    LanePart pt;
    pt.I = 0; pt.beg_b = 0; pt.L_b = 0; pt.tag = 0; pt.r = 0; pt.L = 0; pt.starts = 0u;
    const int N = __reduce_add_sync(kFull, n_b);
    if (N == 0) return pt;
    int I = (N + 31) >> 5, L_b;
    for (;;) {
        // ceil(n_b / I): the fractional part of n_b / I is 0 or >= 1/I >= 1/80, far above the error of the approximate reciprocal
        L_b = (int)((float)n_b * rcp((float)I) + 0.999f);
        if (__reduce_add_sync(kFull, L_b) <= 32) break;
        ++I;
    }
    int x = L_b;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int y = __shfl_up_sync(kFull, x, o);
        if (lane >= o) x += y;
    }
    const int beg_b = x - L_b;
    const unsigned starts = __reduce_or_sync(kFull, L_b > 0 ? (1u << beg_b) : 0u);
    if (L_b > 0) own[beg_b] = tag_b | (L_b << 8) | (beg_b << 16) | (lane << 24); // bits 24+: block lane index
    __syncwarp();
    const int p = 31 - __clz(starts & (kFull >> (31 - lane))); // first lane of this lane's group (bit 0 is always set)
    const int w = own[p];
    __syncwarp();
    pt.I = I; pt.beg_b = beg_b; pt.L_b = L_b; pt.starts = starts;
    pt.tag = w & 0xff; pt.L = (w >> 8) & 0xff;
    pt.r = lane - ((w >> 16) & 0xff);
    return pt;
}

// q-th pair of a block: cs != ct -> (q / nt, q % nt); cs == ct -> q-th pair (lo < hi) of a triangle, from the table
// tri[q] = lo | hi << 8 with q = hi (hi - 1) / 2 + lo.
__device__ __forceinline__ void decode_pair(int q, bool same, int nt, float inv_nt, const uint16_t *__restrict__ tri, int &a, int &b)
{
    if (same) {
        const unsigned w = tri[q];
        a = w & 0xff;
        b = w >> 8;
    } else {
        a = (int)(((float)q + 0.5f) * inv_nt); // (q + 1/2) / nt is at least 1/(2 nt) away from an integer
        b = q - a * nt;
    }
}

// Which centre a warp takes next.  MODE 0: static (warp w takes w, w + W, ...).  MODE 1: one global ticket counter.
// MODE 2: the centres are cut into one contiguous range per SM and the warps of SM s take tickets of range s, so the
// warps that run on one SM at the same time work on ~20 consecutive (cell-sorted) atoms: their neighbour rows and
// positions share L1 lines, and the force reductions that hit the same atom come from one SM instead of queueing
// from many.  A warp whose range is used up moves to any range with centres left, so every centre is processed
// wherever the blocks were placed.  sched[0]: warps that have left (the last one zeroes all counters, so every
// launch starts clean without a memset); sched[32 + s]: tickets taken from range s (MODE 1: s = 0).
#ifndef AEV_FWD_SCHED
#define AEV_FWD_SCHED 1
#endif
#ifndef AEV_BWD_SCHED
#define AEV_BWD_SCHED 4
#endif
// MODE 4 (the reverse kernel): no queue and no persistent grid - a warp takes AEV_CPW consecutive centres and its block
// ends; the hardware's block scheduler levels out the warps.  With the persistent static stride (MODE 0) the warps of the
// 98k-atom water box finished between 217 and 288 us (mean 246 us: the cost of a centre varies with its pair count, and a warp
// keeps its 33 centres whatever they cost); blocks of 4 warps x 2 centres: 0.2915 -> 0.282 ms (4 centres 0.283, 8 0.296,
// one-warp blocks 0.283-0.287).  The ticket queues stay slower for this kernel (0.327 ms, re-measured), also as a hybrid
// (static first, tickets for the last 8-25 %: 0.319-0.332 ms; with an empty ticket phase still 0.35 ms - every warp's centres
// take 22 % longer although the loops compile to the same instructions), and MODE 4 is slower for the forward kernel
// (0.191 against 0.185 ms with tickets).
#ifndef AEV_CPW
#define AEV_CPW 2
#endif
template <int MODE>
struct CentreQueue {
    int *sched;
    int n, nsm, s, lane;
    int beg, end;  // current range
    int pending;   // lane 0: ticket requested and not yet read

    __device__ __forceinline__ void set_range(int r)
    {
        s = r;
        beg = (int)((long long)r * n / nsm);
        end = (int)((long long)(r + 1) * n / nsm);
    }
    __device__ __forceinline__ void init(int *sched_, int n_, int nsm_, int lane_)
    {
        sched = sched_; n = n_; lane = lane_; pending = 0;
        nsm = MODE == 2 ? nsm_ : 1;
        unsigned smid = 0;
        if (MODE == 2) asm("mov.u32 %0, %%smid;" : "=r"(smid));
        set_range((int)(smid % (unsigned)nsm));
    }
    __device__ __forceinline__ void request()
    {
        if (MODE == 4) return;
        if (MODE != 0 && lane == 0) pending = atomicAdd(sched + 32 + s, 1);
    }
    // cur: the centre being processed (MODE 0 only)
    __device__ __forceinline__ int receive(int cur)
    {
        if (MODE == 0) return cur < 0 ? (int)(blockIdx.x * kWarps + (threadIdx.x >> 5)) : cur + (int)(gridDim.x * kWarps);
        if (MODE == 4) { // AEV_CPW consecutive centres per warp, one block after the other (the grid is not persistent)
            if (cur < 0) return (int)(blockIdx.x * kWarps + (threadIdx.x >> 5)) * AEV_CPW;
            return (cur + 1) % AEV_CPW ? cur + 1 : n;
        }
        for (;;) {
            const int t = beg + __shfl_sync(kFull, pending, 0);
            if (t < end) return t;
            if (MODE == 1) return n;
            // range used up: take any range that still has centres (counters only grow, so this terminates)
            int found = -1;
            for (int r0 = 1; r0 < nsm && found < 0; r0 += 32) {
                const int off = r0 + lane;
                int cand = s + off;
                if (cand >= nsm) cand -= nsm;
                bool has = false;
                if (off < nsm) {
                    const int cb = (int)((long long)cand * n / nsm), ce = (int)((long long)(cand + 1) * n / nsm);
                    has = *(volatile int *)(sched + 32 + cand) < ce - cb;
                }
                const unsigned m = __ballot_sync(kFull, has);
                if (m) found = __shfl_sync(kFull, cand, __ffs(m) - 1);
            }
            if (found < 0) return n;
            set_range(found);
            request();
        }
    }
    __device__ __forceinline__ void release()
    {
        if (MODE == 0 || MODE == 4) return;
        int last = 0;
        if (lane == 0) last = atomicAdd(sched, 1) == (int)(gridDim.x * kWarps) - 1;
        if (__shfl_sync(kFull, last, 0)) {
            for (int r = lane; r < nsm; r += 32) atomicExch(sched + 32 + r, 0);
            if (lane == 0) atomicExch(sched, 0);
        }
    }
};

// Everything both kernels do before their arithmetic: lane roles, the segment tables (one centre ahead), the
// radial lane partition, and the batched index / position loads of the current centre.
struct Centre {
    float4 pi;
    LanePart pr;          // radial partition (tag = compact species of this worker lane)
    int wa_beg, wa_end;   // this worker's species segment in the radial row
    int jr[KR];           // radial neighbours of the first KR trips (-1: none)
    float4 xr[KR];
    int ja[KA];           // angular row entries lane + 32 k (-1: none)
    float4 xa[KA];
    int len_a;            // angular row length
    int ab_beg;           // as block lane cs < np: start of the species segment in the angular row
};

__device__ __forceinline__ void load_centre(Centre &c, const AevParams &P, int i, int lane, int my_s, int sgr_l, int sga_l,
                                            const float4 *__restrict__ pos, const int *__restrict__ nbr_r,
                                            const int *__restrict__ nbr_a, int *own)
{
    c.pi = pos[i];
    const int rb_beg = __shfl_sync(kFull, sgr_l, my_s), rb_end = __shfl_sync(kFull, sgr_l, my_s + 1);
    c.ab_beg = __shfl_sync(kFull, sga_l, my_s);
    c.len_a = __shfl_sync(kFull, sga_l, NNP_MAX_SPECIES - 1);
    c.pr = partition(lane < P.np ? rb_end - rb_beg : 0, lane, own, lane);
    c.wa_beg = __shfl_sync(kFull, rb_beg, c.pr.tag);
    c.wa_end = __shfl_sync(kFull, rb_end, c.pr.tag);
    const int *row_r = nbr_r + (size_t)i * P.cap_r;
    const int *row_a = nbr_a + (size_t)i * P.cap_a;
#pragma unroll
    for (int t = 0; t < KR; ++t) {
        const int a = c.wa_beg + c.pr.r + t * c.pr.L;
        c.jr[t] = (c.pr.r < c.pr.L && a < c.wa_end) ? row_r[a] : -1;
    }
#pragma unroll
    for (int k = 0; k < KA; ++k) {
        const int a = lane + 32 * k;
        c.ja[k] = a < c.len_a ? row_a[a] : -1;
    }
#pragma unroll
    for (int t = 0; t < KR; ++t) c.xr[t] = c.jr[t] >= 0 ? pos[c.jr[t]] : c.pi;
#pragma unroll
    for (int k = 0; k < KA; ++k) c.xa[k] = c.ja[k] >= 0 ? pos[c.ja[k]] : c.pi;
}

// Compacts the angular row entries with r < rca into shared memory in row order (= grouped by species); block lane
// cs < np counts the hits in front of its species segment -> seg[].  Returns the count.
template <bool BWD, bool TRIC, class SM>
__device__ __forceinline__ int stage_angular(SM &sm, const AevParams &P, const Centre &c, int i, int lane,
                                             const float4 *__restrict__ pos, const int *__restrict__ nbr_a,
                                             int *__restrict__ flags)
{
    const unsigned lt = (1u << lane) - 1u;
    int na = 0, segc = 0;
    auto chunk = [&](int k, int j, const float4 xj) {
        bool hit = false;
        float3 d = make_float3(0.f, 0.f, 0.f);
        float r2 = 1.f;
        if (j >= 0) {
            d = min_image<TRIC>(c.pi, xj, P);
            r2 = d.x * d.x + d.y * d.y + d.z * d.z;
            hit = r2 < P.rca2;
        }
        const unsigned m = __ballot_sync(kFull, hit);
        if (hit) {
            const int p = na + __popc(m & lt);
            if (p < kCapA) {
                const float rinv = rsq(r2);
                const float r = r2 * rinv;
                float sn, cs_;
                __sincosf(P.pi_rca * r, &sn, &cs_);
                sm.d[p] = make_float4(d.x, d.y, d.z, r);
                // forward: lg2(fc) + 1/2, so that lfc_j + lfc_k = lg2(2 fc_j fc_k) folds the pair prefactor into the
                // exponent of the zeta power; reverse: fc itself
                const float fc = 0.5f * cs_ + 0.5f;
                sm.fr[p] = make_float2(BWD ? fc : lg2(fc) + 0.5f, rinv);
                if constexpr (BWD) {
                    sm.dfc[p] = P.nh_pi_rca * sn;
                    sm.j[p] = j;
                }
            }
        }
        const int bound = c.ab_beg - 32 * k; // entries of this chunk in front of my species segment
        const unsigned below = bound >= 32 ? kFull : (bound <= 0 ? 0u : ((1u << bound) - 1u));
        segc += __popc(m & below);
        na += __popc(m);
    };
#pragma unroll
    for (int k = 0; k < KA; ++k) chunk(k, c.ja[k], c.xa[k]);
    if (c.len_a > 32 * KA) { // rows longer than the prefetched chunks (cap_a > 64)
        const int *row = nbr_a + (size_t)i * P.cap_a;
        for (int k = KA; 32 * k < c.len_a; ++k) {
            const int a = lane + 32 * k;
            const int j = a < c.len_a ? row[a] : -1;
            chunk(k, j, j >= 0 ? pos[j] : c.pi);
        }
    }
    if (na > kCapA) { // more in-cutoff angular neighbours than shared-memory slots
        if (lane == 0) atomicOr(&flags[0], NNP_FLAG_CAP_A);
        na = kCapA;
    }
    if (lane <= NNP_MAX_SPECIES) sm.seg[lane] = lane < P.np ? min(segc, kCapA) : na;
    __syncwarp();
    return na;
}

template <bool LAD, bool TRIC>
__global__ void __launch_bounds__(kWarps * 32, AEV_FWD_MINB)
k_aev_forward(int n, AevParams P, const float4 *__restrict__ pos, const int *__restrict__ nbr_r,
              const uint16_t *__restrict__ seg_r, const int *__restrict__ nbr_a,
              const uint16_t *__restrict__ seg_a, const uint16_t *__restrict__ tri, float *__restrict__ G,
              int *__restrict__ flags, int *__restrict__ sched, int nsm)
{
    __shared__ WarpSmem smem[kWarps];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    // (as in the reverse kernel: an opaque base keeps the compiler from re-deriving it from %tid inside the centre loop -
    // 36 of ~1480 instructions per centre, 0.1853 -> 0.1836 ms)
    uint32_t sm_addr = (uint32_t)__cvta_generic_to_shared(smem) + (uint32_t)wid * (uint32_t)sizeof(WarpSmem);
    asm volatile("mov.b32 %0, %0;" : "+r"(sm_addr));
    WarpSmem &sm = *reinterpret_cast<WarpSmem *>(__cvta_shared_to_generic(sm_addr));
    int bcs, bct;
    block_of_lane(P.np, lane, bcs, bct);
    const int nb_tot = P.np * (P.np + 1) / 2;
    int my_s = 0;
#pragma unroll
    for (int q = 0; q < NNP_MAX_SPECIES - 1; ++q)
        if (lane == q && q < P.np) my_s = P.plist[q];
    // constant factors of the ladder, applied once per feature where lane = feature (1 without ladder)
    const float lad_r = LAD ? P.lad_r[lane & 15] : 1.0f, lad_a = LAD ? P.lad_a[lane >> 2] : 1.0f;

    CentreQueue<AEV_FWD_SCHED> queue;
    queue.init(sched, n, nsm, lane);
    queue.request();
    int i = queue.receive(-1);
    int sgr_l = 0, sga_l = 0;
    if (i < n && lane < NNP_MAX_SPECIES) {
        sgr_l = seg_r[(size_t)i * NNP_MAX_SPECIES + lane];
        sga_l = seg_a[(size_t)i * NNP_MAX_SPECIES + lane];
    }
    while (i < n) {
        queue.request(); // read after the radial phase
        Centre c;
        load_centre(c, P, i, lane, my_s, sgr_l, sga_l, pos, nbr_r, nbr_a, sm.own);
        float *Grow = G + (size_t)i * P.kpad;

        // ---- radial block: G[cs*16+k] = 1/4 sum_j exp(-eta_r (r-ShfR_k)^2) fc(r)
        {
            float2 acc[NNP_NSHF_R / 2];
#pragma unroll
            for (int k = 0; k < NNP_NSHF_R / 2; ++k) acc[k] = make_float2(0.f, 0.f);
            auto term = [&](const float4 xj) {
                const float3 d = min_image<TRIC>(c.pi, xj, P);
                const float r2 = d.x * d.x + d.y * d.y + d.z * d.z;
                if (r2 < P.rcr2) {
                    const float r = r2 * rsq(r2);
                    const float2 fc = bc2(0.125f * __cosf(P.pi_rcr * r) + 0.125f); // (1/4) fc
                    const float2 u = bc2(P.kr * r);
                    if constexpr (LAD) {
                        // anchors k = 1, 5, 9, 13; acc[2m] = shifts (4m, 4m+1), acc[2m+1] = (4m+2, 4m+3), unscaled
                        float2 t[NNP_NSHF_R / 8];
#pragma unroll
                        for (int mp = 0; mp < NNP_NSHF_R / 8; ++mp) {
                            const float2 w = add2(u, P.nkr_anc2[mp]);
                            const float2 ww = mul2(w, w);
                            t[mp] = mul2(fc, make_float2(ex2(-ww.x), ex2(-ww.y)));
                        }
                        const float x = P.two_dlt_r * (u.x - P.kr_shf[1]);
                        const float q = ex2(x);
                        const float2 pq0 = make_float2(ex2(-x), 1.0f), pq1 = make_float2(q, q * q);
#pragma unroll
                        for (int mp = 0; mp < NNP_NSHF_R / 8; ++mp) {
                            acc[4 * mp] = fma2(bc2(t[mp].x), pq0, acc[4 * mp]);
                            acc[4 * mp + 1] = fma2(bc2(t[mp].x), pq1, acc[4 * mp + 1]);
                            acc[4 * mp + 2] = fma2(bc2(t[mp].y), pq0, acc[4 * mp + 2]);
                            acc[4 * mp + 3] = fma2(bc2(t[mp].y), pq1, acc[4 * mp + 3]);
                        }
                    } else {
#pragma unroll
                        for (int k = 0; k < NNP_NSHF_R / 2; ++k) {
                            const float2 w = add2(u, P.nkr_shf2[k]);
                            const float2 ww = mul2(w, w);
                            acc[k] = fma2(fc, make_float2(ex2(-ww.x), ex2(-ww.y)), acc[k]);
                        }
                    }
                }
            };
#pragma unroll
            for (int t = 0; t < KR; ++t)
                if (c.jr[t] >= 0) term(c.xr[t]);
            if (c.pr.I > KR) {
                const int *row = nbr_r + (size_t)i * P.cap_r;
                for (int t = KR; t < c.pr.I; ++t) {
                    const int a = c.wa_beg + c.pr.r + t * c.pr.L;
                    if (c.pr.r < c.pr.L && a < c.wa_end) term(pos[row[a]]);
                }
            }
            if (c.pr.I > 0) {
                float *myrow = sm.red + lane * kRedLd;
#pragma unroll
                for (int q4 = 0; q4 < NNP_NSHF_R / 4; ++q4)
                    *reinterpret_cast<float4 *>(myrow + 4 * q4) = make_float4(acc[2 * q4].x, acc[2 * q4].y, acc[2 * q4 + 1].x, acc[2 * q4 + 1].y);
                __syncwarp();
            }
            // rows [beg_b, beg_b + L_b) belong to species b; a half warp sums the 16 columns of one species
            for (int p0 = 0; p0 < P.np; p0 += 2) {
                const int cs = p0 + (lane >> 4);
                const int csc = min(cs, P.np - 1);
                const int beg = __shfl_sync(kFull, c.pr.beg_b, csc);
                int L = __shfl_sync(kFull, c.pr.L_b, csc);
                if (cs >= P.np) L = 0;
                float sum = 0.f;
                for (int rr = beg; rr < beg + L; ++rr) sum += sm.red[rr * kRedLd + (lane & 15)];
                if (cs < P.np) Grow[cs * NNP_NSHF_R + (lane & 15)] = sum * lad_r;
            }
            for (int q = P.aev_len + lane; q < P.kpad; q += 32) Grow[q] = 0.f; // zero padding columns
            __syncwarp();
        }

        // ---- angular block
        const int i_next = queue.receive(i);
        int sgr_n = 0, sga_n = 0; // segment tables of the next centre
        if (i_next < n && lane < NNP_MAX_SPECIES) {
            sgr_n = seg_r[(size_t)i_next * NNP_MAX_SPECIES + lane];
            sga_n = seg_a[(size_t)i_next * NNP_MAX_SPECIES + lane];
        }
        stage_angular<false, TRIC>(sm, P, c, i, lane, pos, nbr_a, flags);
        int n_b = 0;
        if (lane < nb_tot) {
            const int ns = sm.seg[bcs + 1] - sm.seg[bcs], nt = sm.seg[bct + 1] - sm.seg[bct];
            n_b = bcs == bct ? ns * (ns - 1) / 2 : ns * nt;
        }
        const LanePart pt = partition(n_b, bcs | (bct << 3), sm.own, lane);
        // blocks without a pair are zero rows of G
        for (unsigned zm = __ballot_sync(kFull, lane < nb_tot && n_b == 0); zm; zm &= zm - 1)
            Grow[P.n_rad + (__ffs(zm) - 1) * NNP_ANG_BLOCK + lane] = 0.f;
        if (pt.I > 0) {
            float2 acc[NNP_ANG_BLOCK / 2]; // [a][z pair]
#pragma unroll
            for (int q = 0; q < NNP_ANG_BLOCK / 2; ++q) acc[q] = make_float2(0.f, 0.f);
            const int wcs = pt.tag & 7, wct = pt.tag >> 3;
            const int a0 = sm.seg[wcs], b0 = sm.seg[wct];
            const int nt = sm.seg[wct + 1] - b0;
            const bool same = wcs == wct;
            int npairs = 0;
            if (pt.r < pt.L) {
                const int ns = sm.seg[wcs + 1] - a0;
                npairs = same ? ns * (ns - 1) / 2 : ns * nt;
            }
            const float inv_nt = rcp((float)max(nt, 1));
            const float2 zeta2 = bc2(P.zeta), half2 = bc2(0.5f);
            for (int q = pt.r; q < npairs; q += pt.L) {
                int ia, ib;
                decode_pair(q, same, nt, inv_nt, tri, ia, ib);
                ia += a0; ib += same ? a0 : b0;
                const float4 dj = sm.d[ia], dk = sm.d[ib];
                const float2 fj = sm.fr[ia], fk = sm.fr[ib]; // (lg2 fc + 1/2, 1/r)
                const float lff = fj.x + fk.x;               // lg2(2 fc_j fc_k)
                const float cc = (0.95f * fj.y * fk.y) * (dj.x * dk.x + dj.y * dk.y + dj.z * dk.z);
                const float s2 = fmaf(-cc, cc, 1.0f);
                const float sn = s2 * rsq(s2);
                const float2 cc2 = bc2(cc), sn2 = bc2(sn), lff2 = bc2(lff);
                // F_z = 2 fc_j fc_k ((1 + cos(theta' - ShfZ_z)) / 2)^zeta = 2^(zeta lg2(base_z) + lff)
                float2 fz[NNP_NSHF_Z / 2];
#pragma unroll
                for (int zp = 0; zp < NNP_NSHF_Z / 2; ++zp) {
                    const float2 base = fma2(cc2, P.hcz2[zp], fma2(sn2, P.hsz2[zp], half2));
                    const float2 e = fma2(zeta2, make_float2(lg2(base.x), lg2(base.y)), lff2);
                    fz[zp] = make_float2(ex2(e.x), ex2(e.y));
                }
                const float2 u = bc2(P.half_ka * (dj.w + dk.w));
                float2 ra[NNP_NSHF_A / 2]; // radial factors (a, a+1); with the ladder: without their constant factors
                if constexpr (LAD) {
                    const float2 w = add2(u, P.nka_anc2); // anchors a = 1, 5
                    const float2 ww = mul2(w, w);
                    const float x = P.two_dlt_a * w.x;
                    const float q = ex2(x);
                    const float2 pq0 = make_float2(ex2(-x), 1.0f), pq1 = make_float2(q, q * q);
                    const float e0 = ex2(-ww.x), e1 = ex2(-ww.y);
                    ra[0] = mul2(bc2(e0), pq0); ra[1] = mul2(bc2(e0), pq1);
                    ra[2] = mul2(bc2(e1), pq0); ra[3] = mul2(bc2(e1), pq1);
                } else {
#pragma unroll
                    for (int ap = 0; ap < NNP_NSHF_A / 2; ++ap) {
                        const float2 w = add2(u, P.nka_shf2[ap]);
                        const float2 ww = mul2(w, w);
                        ra[ap] = make_float2(ex2(-ww.x), ex2(-ww.y));
                    }
                }
#pragma unroll
                for (int ap = 0; ap < NNP_NSHF_A / 2; ++ap) {
#pragma unroll
                    for (int zp = 0; zp < NNP_NSHF_Z / 2; ++zp) {
                        acc[(2 * ap) * 2 + zp] = fma2(bc2(ra[ap].x), fz[zp], acc[(2 * ap) * 2 + zp]);
                        acc[(2 * ap + 1) * 2 + zp] = fma2(bc2(ra[ap].y), fz[zp], acc[(2 * ap + 1) * 2 + zp]);
                    }
                }
            }
            float *myrow = sm.red + lane * kRedLd;
#pragma unroll
            for (int q4 = 0; q4 < NNP_ANG_BLOCK / 4; ++q4)
                *reinterpret_cast<float4 *>(myrow + 4 * q4) = make_float4(acc[2 * q4].x, acc[2 * q4].y, acc[2 * q4 + 1].x, acc[2 * q4 + 1].y);
            __syncwarp();
            // Rows of the transpose buffer are grouped by block (lane groups of the partition; lanes past the last
            // group hold zeros).  lane = feature inside the block: one running sum over the 32 rows, flushed as one
            // coalesced 128 B store wherever the next row starts a new group (warp-uniform branches).
            float sum = 0.f;
            float *gp = Grow + P.n_rad + lane + (sm.own[0] >> 24) * NNP_ANG_BLOCK; // block lane index = block index p
#pragma unroll
            for (int rr = 0; rr < 32; ++rr) {
                sum += sm.red[rr * kRedLd + lane];
                if (rr == 31 || (pt.starts >> (rr + 1) & 1u)) {
                    *gp = sum * lad_a;
                    sum = 0.f;
                    if (rr < 31) gp = Grow + P.n_rad + lane + (sm.own[rr + 1] >> 24) * NNP_ANG_BLOCK;
                }
            }
        }
        __syncwarp();
        sgr_l = sgr_n; sga_l = sga_n;
        i = i_next;
    }
    queue.release();
}

// Reverse pass: g = dE/dG_i (row of dG, times inv_nets).  Adds -dE/dx to frc for the centre and its neighbours.
// (The Gaussian ladder of the forward kernel is not used here: the reverse pass needs every w_k as well, the
// recurrence then costs more issue slots than the exponentials it saves -- measured 0.355 vs 0.346 ms.)
// GS: the centre's gradient row (kpad <= kGsMax floats) is copied into shared memory with cp.async at the top of the
// iteration, behind the index -> position load chain, instead of being loaded from global memory where it is first
// needed (those loads were 10 % of the stall samples).
constexpr int kGsMax = 128;  // water: 128 active columns; 2 KiB per block keeps five blocks per SM
// VIR: also accumulate the virial V_ab = sum_d d_a (dE/dd)_b over every displacement vector the energy is built from
// (PAPER.md L262): six per-lane sums over all centres of the warp, reduced once at the end.
template <bool GS, bool VIR, bool TRIC>
__global__ void __launch_bounds__(kWarps * 32, AEV_BWD_MINB)
k_aev_backward(int n, AevParams P, const float4 *__restrict__ pos, const int *__restrict__ nbr_r,
               const uint16_t *__restrict__ seg_r, const int *__restrict__ nbr_a,
               const uint16_t *__restrict__ seg_a, const uint16_t *__restrict__ tri, const float *__restrict__ dG,
               float inv_nets, float4 *__restrict__ frc, int *__restrict__ flags, int *__restrict__ sched, int nsm,
               double *__restrict__ virial /* [6] xx yy zz xy xz yz, VIR only */)
{
    extern __shared__ __align__(16) uint8_t smem_dyn[];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    // The warp's shared-memory base is made opaque to the compiler: left alone it re-derives the address from
    // %tid / the shared window (two S2R + four ALU instructions) inside every trip of the pair loop.
    uint32_t sm_addr = (uint32_t)__cvta_generic_to_shared(smem_dyn) + (uint32_t)wid * (uint32_t)sizeof(WarpSmemBwd);
    asm volatile("mov.b32 %0, %0;" : "+r"(sm_addr));
    WarpSmemBwd &sm = *reinterpret_cast<WarpSmemBwd *>(__cvta_shared_to_generic(sm_addr));
    float *gs = reinterpret_cast<float *>(smem_dyn + kWarps * sizeof(WarpSmemBwd)) + wid * kGsMax; // GS only
    int bcs, bct;
    block_of_lane(P.np, lane, bcs, bct);
    const int nb_tot = P.np * (P.np + 1) / 2;
    int my_s = 0;
#pragma unroll
    for (int q = 0; q < NNP_MAX_SPECIES - 1; ++q)
        if (lane == q && q < P.np) my_s = P.plist[q];
    // P.k_ang0 = zeta 0.95 (hcz2 / hsz2 carry the 1/2 of the base); d/drb exp(-eta (rb - s)^2) = -2 eta (rb - s) ra =
    // (-2 eta / ka) w ra with w = ka (rb - s): P.half_drb_scale, P.dr_scale (AevParams, nnp_aev_derive)
    float (*fsm)[3] = reinterpret_cast<float (*)[3]>(sm.ab);

    // Centres are assigned statically, AEV_CPW consecutive ones per warp of a non-persistent grid (AEV_BWD_SCHED 4, above);
    // for this kernel the ticket queues measured slower, see DESIGN.md section 6.
    float vir[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    CentreQueue<AEV_BWD_SCHED> queue;
    queue.init(sched, n, nsm, lane);
    queue.request();
    int i = queue.receive(-1);
    int sgr_l = 0, sga_l = 0;
    if (i < n && lane < NNP_MAX_SPECIES) {
        sgr_l = seg_r[(size_t)i * NNP_MAX_SPECIES + lane];
        sga_l = seg_a[(size_t)i * NNP_MAX_SPECIES + lane];
    }
    while (i < n) {
        queue.request(); // read after the radial phase
        if constexpr (GS) {
            const float *src = dG + (size_t)i * P.kpad;
            for (int q = 4 * lane; q < P.kpad; q += 128)
                asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(gs + q)), "l"(src + q) : "memory");
            asm volatile("cp.async.commit_group;" ::: "memory");
        }
        Centre c;
        load_centre(c, P, i, lane, my_s, sgr_l, sga_l, pos, nbr_r, nbr_a, sm.own);
        const float *grow = dG + (size_t)i * P.kpad;
        auto g4 = [&](int off) -> float4 { // four gradient values of this centre (off: multiple of 4)
            if constexpr (GS) return *reinterpret_cast<const float4 *>(gs + off);
            else return *reinterpret_cast<const float4 *>(grow + off);
        };
        if constexpr (GS) {
            asm volatile("cp.async.wait_all;" ::: "memory");
            __syncwarp();
        }
        float fi[3] = {0.f, 0.f, 0.f}; // dE/dd summed over this lane's terms (force on i = +sum)

        // ---- radial: dE/dr_ij = sum_k g[s_j*16+k] * 1/4 e_k (-2 eta (r-ShfR_k) fc + fc')
        if (c.pr.I > 0) {
            float2 gr[NNP_NSHF_R / 2];
            const float scr = 0.25f * inv_nets; // the 1/4 of the radial term and 1 / n_nets scale dE/dr once, not the 16 gradients
#pragma unroll
            for (int k4 = 0; k4 < NNP_NSHF_R / 4; ++k4) {
                float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
                if (c.pr.r < c.pr.L) v = g4(c.pr.tag * NNP_NSHF_R + 4 * k4);
                gr[2 * k4] = make_float2(v.x, v.y);
                gr[2 * k4 + 1] = make_float2(v.z, v.w);
            }
            auto term = [&](int j, const float4 xj) {
                const float3 d = min_image<TRIC>(c.pi, xj, P);
                const float r2 = d.x * d.x + d.y * d.y + d.z * d.z;
                if (r2 < P.rcr2) {
                    const float rinv = rsq(r2);
                    const float r = r2 * rinv;
                    float sn, cs_;
                    __sincosf(P.pi_rcr * r, &sn, &cs_);
                    const float2 fc = bc2((0.5f * cs_ + 0.5f) * P.dr_scale);
                    const float2 dfc = bc2(P.nh_pi_rcr * sn);
                    const float2 u = bc2(P.kr * r);
                    float2 acc = make_float2(0.f, 0.f);
#pragma unroll
                    for (int k = 0; k < NNP_NSHF_R / 2; ++k) {
                        const float2 w = add2(u, P.nkr_shf2[k]);
                        const float2 ww = mul2(w, w);
                        const float2 e = make_float2(ex2(-ww.x), ex2(-ww.y));
                        acc = fma2(mul2(gr[k], e), fma2(w, fc, dfc), acc);
                    }
                    const float dEdr = acc.x + acc.y;
                    const float sc = dEdr * (rinv * scr);
                    const float vx = sc * d.x, vy = sc * d.y, vz = sc * d.z;
                    atomicAdd(&frc[j], make_float4(-vx, -vy, -vz, 0.f));
                    fi[0] += vx; fi[1] += vy; fi[2] += vz;
                    if constexpr (VIR) {
                        vir[0] = fmaf(d.x, vx, vir[0]); vir[1] = fmaf(d.y, vy, vir[1]); vir[2] = fmaf(d.z, vz, vir[2]);
                        vir[3] = fmaf(d.x, vy, vir[3]); vir[4] = fmaf(d.x, vz, vir[4]); vir[5] = fmaf(d.y, vz, vir[5]);
                    }
                }
            };
#pragma unroll
            for (int t = 0; t < KR; ++t)
                if (c.jr[t] >= 0) term(c.jr[t], c.xr[t]);
            if (c.pr.I > KR) {
                const int *row = nbr_r + (size_t)i * P.cap_r;
                for (int t = KR; t < c.pr.I; ++t) {
                    const int a = c.wa_beg + c.pr.r + t * c.pr.L;
                    if (c.pr.r < c.pr.L && a < c.wa_end) { const int j = row[a]; term(j, pos[j]); }
                }
            }
        }

        // ---- angular
        const int i_next = queue.receive(i);
        int sgr_n = 0, sga_n = 0; // segment tables of the next centre
        if (i_next < n && lane < NNP_MAX_SPECIES) {
            sgr_n = seg_r[(size_t)i_next * NNP_MAX_SPECIES + lane];
            sga_n = seg_a[(size_t)i_next * NNP_MAX_SPECIES + lane];
        }
        const int na = stage_angular<true, TRIC>(sm, P, c, i, lane, pos, nbr_a, flags);
        const bool arena = na <= kMat; // warp-uniform
        if (arena) {
            if (lane < na) sm.ab[lane * kMatLd + lane] = make_float2(0.f, 0.f);
        } else {
            for (int a = lane; a < na; a += 32) { fsm[a][0] = 0.f; fsm[a][1] = 0.f; fsm[a][2] = 0.f; }
        }
        __syncwarp();
        int n_b = 0;
        if (lane < nb_tot) {
            const int ns = sm.seg[bcs + 1] - sm.seg[bcs], nt = sm.seg[bct + 1] - sm.seg[bct];
            n_b = bcs == bct ? ns * (ns - 1) / 2 : ns * nt;
        }
        const LanePart pt = partition(n_b, bcs | (bct << 3), sm.own, lane);
        if (pt.I > 0) {
            const int wcs = pt.tag & 7, wct = pt.tag >> 3;
            const int a0 = sm.seg[wcs], b0 = sm.seg[wct];
            const int nt = sm.seg[wct + 1] - b0;
            const bool same = wcs == wct;
            int npairs = 0;
            if (pt.r < pt.L) {
                const int ns = sm.seg[wcs + 1] - a0;
                npairs = same ? ns * (ns - 1) / 2 : ns * nt;
            }
            const float inv_nt = rcp((float)max(nt, 1));
            float2 gw[NNP_ANG_BLOCK / 2]; // [a][z pair]
            {
                const int pb = wcs * (2 * P.np + 1 - wcs) / 2 + (wct - wcs);
                const int gp = P.n_rad + pb * NNP_ANG_BLOCK;
#pragma unroll
                for (int q4 = 0; q4 < NNP_ANG_BLOCK / 4; ++q4) {
                    float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (npairs > 0) v = g4(gp + 4 * q4);
                    gw[2 * q4] = make_float2(v.x, v.y);
                    gw[2 * q4 + 1] = make_float2(v.z, v.w);
                }
            }
            const float2 zm12 = bc2(P.zm1), half2 = bc2(0.5f);
            const float sc_ang = 2.0f * inv_nets;
            for (int q = pt.r; q < npairs; q += pt.L) {
                int ia, ib;
                decode_pair(q, same, nt, inv_nt, tri, ia, ib);
                ia += a0; ib += same ? a0 : b0;
                const float4 dj = sm.d[ia], dk = sm.d[ib];
                const float2 fj = sm.fr[ia], fk = sm.fr[ib];
                const float rjk_inv = fj.y * fk.y;
                const float cs_ = (dj.x * dk.x + dj.y * dk.y + dj.z * dk.z) * rjk_inv; // cos(theta)
                const float cc = 0.95f * cs_;
                const float s2 = fmaf(-cc, cc, 1.0f);
                const float sn_inv = rsq(s2);
                const float sn = s2 * sn_inv;
                const float2 cc2 = bc2(cc), sn2 = bc2(sn);
                float2 fz[NNP_NSHF_Z / 2], dfz[NNP_NSHF_Z / 2]; // F_z and (dF_z/dcos(theta)) / k_ang
#pragma unroll
                for (int zp = 0; zp < NNP_NSHF_Z / 2; ++zp) {
                    const float2 hc = P.hcz2[zp];
                    const float2 base = fma2(cc2, hc, fma2(sn2, P.hsz2[zp], half2));
                    const float2 e = mul2(zm12, make_float2(lg2(base.x), lg2(base.y)));
                    const float2 pw = make_float2(ex2(e.x), ex2(e.y)); // base^(zeta-1)
                    fz[zp] = mul2(pw, base);
                    // dF/dtheta' = -(zeta/2) sin(theta'-phi) base^(zeta-1); dtheta'/dcos = -0.95/sn
                    dfz[zp] = mul2(fma2(sn2, hc, mul2(cc2, P.nhsz2[zp])), pw);
                }
                // A_z = sum_a g[a][z] ra_a (value and angular derivative), C_z = sum_a g[a][z] ra_a w_a (radial derivative)
                float2 Az[NNP_NSHF_Z / 2], Cz[NNP_NSHF_Z / 2];
#pragma unroll
                for (int zp = 0; zp < NNP_NSHF_Z / 2; ++zp) { Az[zp] = make_float2(0.f, 0.f); Cz[zp] = make_float2(0.f, 0.f); }
                const float2 u = bc2(P.half_ka * (dj.w + dk.w));
#pragma unroll
                for (int ap = 0; ap < NNP_NSHF_A / 2; ++ap) {
                    const float2 w = add2(u, P.nka_shf2[ap]);
                    const float2 ww = mul2(w, w);
                    const float2 ra = make_float2(ex2(-ww.x), ex2(-ww.y));
                    const float2 rw = mul2(ra, w);
#pragma unroll
                    for (int zp = 0; zp < NNP_NSHF_Z / 2; ++zp) {
                        Az[zp] = fma2(gw[(2 * ap) * 2 + zp], bc2(ra.x), Az[zp]);
                        Cz[zp] = fma2(gw[(2 * ap) * 2 + zp], bc2(rw.x), Cz[zp]);
                        Az[zp] = fma2(gw[(2 * ap + 1) * 2 + zp], bc2(ra.y), Az[zp]);
                        Cz[zp] = fma2(gw[(2 * ap + 1) * 2 + zp], bc2(rw.y), Cz[zp]);
                    }
                }
                const float2 T2 = fma2(Az[0], fz[0], mul2(Az[1], fz[1]));
                const float2 D2 = fma2(Az[0], dfz[0], mul2(Az[1], dfz[1]));
                const float2 R2 = fma2(Cz[0], fz[0], mul2(Cz[1], fz[1]));
                const float T = (T2.x + T2.y) * sc_ang; // (the prefactor 2 and 1 / n_nets scale the three sums, not the 32 gradients)
                float dE_dcs = D2.x + D2.y;
                const float dE_drb = R2.x + R2.y;
                const float ff = (fj.x * fk.x) * sc_ang;
                dE_dcs *= ff * (P.k_ang0 * sn_inv);
                const float half_drb = P.half_drb_scale * dE_drb * ff;
                const float dE_drj = fmaf(T * sm.dfc[ia], fk.x, half_drb);
                const float dE_drk = fmaf(T * fj.x, sm.dfc[ib], half_drb);
                const float beta = dE_dcs * rjk_inv;
                const float alj = (dE_drj - dE_dcs * cs_ * fj.y) * fj.y;
                const float alk = (dE_drk - dE_dcs * cs_ * fk.y) * fk.y;
                if (arena) {
                    const int sab = ia * kMatLd + ib, sba = ib * kMatLd + ia;
                    sm.ab[sab] = make_float2(alj, beta);
                    sm.ab[sba] = make_float2(alk, beta);
                } else {
                    atomicAdd(&fsm[ia][0], alj * dj.x + beta * dk.x);
                    atomicAdd(&fsm[ia][1], alj * dj.y + beta * dk.y);
                    atomicAdd(&fsm[ia][2], alj * dj.z + beta * dk.z);
                    atomicAdd(&fsm[ib][0], beta * dj.x + alk * dk.x);
                    atomicAdd(&fsm[ib][1], beta * dj.y + alk * dk.y);
                    atomicAdd(&fsm[ib][2], beta * dj.z + alk * dk.z);
                }
            }
        }
        __syncwarp();
        // second pass: lane = neighbour a; dE/dd_a = sum_b (alpha_a(ab) d_a + beta(ab) d_b)
        for (int a = lane; a < na; a += 32) {
            float fx, fy, fz;
            if (arena) {
                const float4 da = sm.d[a];
                float asum = 0.f;
                fx = 0.f; fy = 0.f; fz = 0.f;
                const float2 *rab = sm.ab + a * kMatLd;
                for (int b = 0; b < na; ++b) {
                    const float2 w = rab[b];
                    const float4 db = sm.d[b];
                    asum += w.x;
                    fx = fmaf(w.y, db.x, fx); fy = fmaf(w.y, db.y, fy); fz = fmaf(w.y, db.z, fz);
                }
                fx = fmaf(asum, da.x, fx); fy = fmaf(asum, da.y, fy); fz = fmaf(asum, da.z, fz);
            } else {
                fx = fsm[a][0]; fy = fsm[a][1]; fz = fsm[a][2];
            }
            atomicAdd(&frc[sm.j[a]], make_float4(-fx, -fy, -fz, 0.f));
            fi[0] += fx; fi[1] += fy; fi[2] += fz;
            if constexpr (VIR) {
                const float4 dv = sm.d[a];
                vir[0] = fmaf(dv.x, fx, vir[0]); vir[1] = fmaf(dv.y, fy, vir[1]); vir[2] = fmaf(dv.z, fz, vir[2]);
                vir[3] = fmaf(dv.x, fy, vir[3]); vir[4] = fmaf(dv.x, fz, vir[4]); vir[5] = fmaf(dv.y, fz, vir[5]);
            }
        }
#pragma unroll
        for (int q = 0; q < 3; ++q) {
#pragma unroll
            for (int o = 16; o >= 1; o >>= 1) fi[q] += __shfl_xor_sync(kFull, fi[q], o);
        }
        if (lane == 0) atomicAdd(&frc[i], make_float4(fi[0], fi[1], fi[2], 0.f));
        __syncwarp();
        sgr_l = sgr_n; sga_l = sga_n;
        i = i_next;
    }
    queue.release();
    if constexpr (VIR) {
#pragma unroll
        for (int q = 0; q < 6; ++q) {
            double v = (double)vir[q];
#pragma unroll
            for (int o = 16; o >= 1; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
            if (lane == 0) atomicAdd(virial + q, v);
        }
    }
}

int g_blocks_fwd = 0, g_sms = 0;

} // namespace

// tri[q] = lo | hi << 8 for the q-th pair (lo < hi) of a triangle, q = hi (hi - 1) / 2 + lo, hi < kCapA
void nnp_aev_tri_table(uint16_t *h_tri /* [NNP_TRI_LEN] */)
{
    int q = 0;
    for (int hi = 1; hi < kCapA; ++hi)
        for (int lo = 0; lo < hi; ++lo) h_tri[q++] = (uint16_t)(lo | (hi << 8));
}

static int persistent_grid(nnp_ctx *c, int blocks_per_sm)
{
    if (!g_sms) {
        cudaDeviceGetAttribute(&g_sms, cudaDevAttrMultiProcessorCount, c->device);
        if (g_sms <= 0) g_sms = 148;
        if (g_sms > 1024) g_sms = 1024;
    }
    const int want = nnp_div_up(c->n, kWarps);
    const int cap = g_sms * (blocks_per_sm > 0 ? blocks_per_sm : 1);
    return want < cap ? want : cap;
}

void nnp_launch_aev_forward(nnp_ctx *c)
{
    if (!g_blocks_fwd) cudaOccupancyMaxActiveBlocksPerMultiprocessor(&g_blocks_fwd, k_aev_forward<true, false>, kWarps * 32, 0);
    const int grid = persistent_grid(c, g_blocks_fwd);
    auto kern = c->aev.tric ? (c->aev.ladder ? k_aev_forward<true, true> : k_aev_forward<false, true>)
                            : (c->aev.ladder ? k_aev_forward<true, false> : k_aev_forward<false, false>);
    kern<<<grid, kWarps * 32, 0, c->stream>>>(c->n, c->aev, c->pos, c->nbr_r, c->seg_r, c->nbr_a,
                                                                                  c->seg_a, c->d_tri, c->G, c->flags, c->aev_sched, g_sms);
    c->launches += 1;
}

void nnp_launch_aev_backward(nnp_ctx *c, float inv_nets, double *d_virial)
{
    const int gs = c->aev.kpad <= kGsMax ? 1 : 0, vir = d_virial ? 1 : 0;
    const int smem = (int)sizeof(WarpSmemBwd) * kWarps + (gs ? kWarps * kGsMax * 4 : 0);
    static int blocks[2][2] = {{0, 0}, {0, 0}};
    auto kern = c->aev.tric ? (gs ? (vir ? k_aev_backward<true, true, true> : k_aev_backward<true, false, true>)
                                  : (vir ? k_aev_backward<false, true, true> : k_aev_backward<false, false, true>))
                            : (gs ? (vir ? k_aev_backward<true, true, false> : k_aev_backward<true, false, false>)
                                  : (vir ? k_aev_backward<false, true, false> : k_aev_backward<false, false, false>));
    if (!blocks[gs][vir]) {
        cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&blocks[gs][vir], kern, kWarps * 32, smem);
    }
    const int grid = AEV_BWD_SCHED == 4 ? nnp_div_up(c->n, kWarps * AEV_CPW) : persistent_grid(c, blocks[gs][vir]);
    kern<<<grid, kWarps * 32, smem, c->stream>>>(
        c->n, c->aev, c->pos, c->nbr_r, c->seg_r, c->nbr_a, c->seg_a, c->d_tri, c->dG, inv_nets, c->frc, c->flags, c->aev_sched + NNP_AEV_SCHED_LEN, g_sms,
        d_virial);
    c->launches += 1;
}
