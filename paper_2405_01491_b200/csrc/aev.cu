// Stage 2 (AEV forward) and the AEV half of stage 4 (reverse pass + force scatter).
// Definition: SURVEY.md 8(c) O2/O3/O6 (PAPER.md L61 cosine switch, L79 Gaussian radial basis, L443 angular form
// (0.5+0.5cos(theta-theta_n))^zeta, L55 pairs of edges with a common centre, L65/L176 forces by reverse mode).
//
// One warp per centre atom.  Neighbour rows are grouped by neighbour species (stage 1), so
//   radial:  lane = neighbour, 16 Gaussians in registers per species segment, butterfly reduction over lanes;
//   angular: the in-cutoff neighbours are compacted into shared memory (dx,dy,dz,r | fc | fc'), then for each
//            non-empty species pair (s,t) lanes take pairs (j,k), keep the 8x4 terms in 32 registers and a
//            31-shuffle butterfly leaves feature `lane` of that 32-wide block in lane `lane` -> one coalesced
//            128 B store.  Triplets are enumerated on the fly and never stored (the paper's
//            GraphAngularExtension stores them, L55).
//   reverse: per pair only three scalars (alpha_j, alpha_k, beta with dE/dd_ij = alpha_j d_ij + beta d_ik) are
//            parked in a per-warp shared-memory arena; a second pass with lane = neighbour sums them into the
//            neighbour forces without atomics; one 16-byte vector reduction per neighbour goes to global.
// cos(theta' - ShfZ) with theta' = acos(0.95 cos theta) is expanded as c' cos ShfZ + sqrt(1-c'^2) sin ShfZ: no acos.
#include "nnp_internal.cuh"

namespace {

constexpr int kWarps = 4;
constexpr int kCapA = 64;        // shared-memory slots for in-cutoff angular neighbours per centre
constexpr int kArena = 704;      // pair records per warp: covers n <= 38 in-cutoff neighbours (703 pairs)

struct WarpSmem {
    float4 d[kCapA];   // dx, dy, dz, r
    float fc[kCapA];
    int seg[NNP_MAX_SPECIES + 1];
};
struct WarpSmemBwd {
    float4 d[kCapA];
    float fc[kCapA];
    float dfc[kCapA];
    float f[kCapA][3]; // dE/dd per neighbour (fallback path accumulates here with atomics)
    int j[kCapA];
    int seg[NNP_MAX_SPECIES + 1];
    float alo[kArena], ahi[kArena], bet[kArena]; // pair (a<b): alpha of a, alpha of b, beta
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

__device__ __forceinline__ float3 min_image(const float4 a, const float4 b, const AevParams &P)
{
    float dx = b.x - a.x, dy = b.y - a.y, dz = b.z - a.z;
    if (P.periodic) {
        dx -= P.box[0] * rintf(dx * P.inv_box[0]);
        dy -= P.box[1] * rintf(dy * P.inv_box[1]);
        dz -= P.box[2] * rintf(dz * P.inv_box[2]);
    }
    return make_float3(dx, dy, dz);
}

// Sum v[0..N) over the 32 lanes; afterwards lane l holds in v[0] the total of element (l >> (5 - log2 N)).
template <int N>
__device__ __forceinline__ void butterfly_reduce(float (&v)[N], int lane)
{
    static_assert(N == 16 || N == 32, "N");
    int w = 16;
#pragma unroll
    for (int m = N / 2; m >= 1; m >>= 1, w >>= 1) {
        const bool upper = lane & w;
#pragma unroll
        for (int q = 0; q < m; ++q) {
            float send = upper ? v[q] : v[q + m];
            float keep = upper ? v[q + m] : v[q];
            v[q] = keep + __shfl_xor_sync(0xffffffffu, send, w);
        }
    }
    if (N == 16) v[0] += __shfl_xor_sync(0xffffffffu, v[0], 1);
}

// Compacts the angular neighbours with r < rca into shared memory, keeping the species grouping.
// Returns the count; *present gets one bit per species with at least one in-cutoff neighbour.
template <bool BWD, class SM>
__device__ __forceinline__ int stage_angular(SM &sm, const AevParams &P, int i, int lane, const float4 pi,
                                             const float4 *__restrict__ pos, const int *__restrict__ nbr_a,
                                             const uint16_t *__restrict__ seg_a, int *__restrict__ flags,
                                             unsigned *present)
{
    const uint16_t *sg = seg_a + (size_t)i * NNP_MAX_SPECIES;
    const int *row = nbr_a + (size_t)i * P.cap_a;
    const unsigned lt = (1u << lane) - 1u;
    int na = 0;
    unsigned pm = 0;
    for (int s = 0; s < P.S; ++s) {
        if (lane == 0) sm.seg[s] = na;
        const int a_beg = sg[s], a_end = sg[s + 1];
        const int na0 = na;
        for (int a0 = a_beg; a0 < a_end; a0 += 32) {
            const int a = a0 + lane;
            bool hit = false;
            float3 d = make_float3(0.f, 0.f, 0.f);
            float r2 = 0.f;
            int j = 0;
            if (a < a_end) {
                j = row[a];
                d = min_image(pi, pos[j], P);
                r2 = d.x * d.x + d.y * d.y + d.z * d.z;
                hit = r2 < P.rca2;
            }
            const unsigned m = __ballot_sync(0xffffffffu, hit);
            if (hit) {
                const int p = na + __popc(m & lt);
                if (p < kCapA) {
                    const float rinv = rsqrtf(r2);
                    const float r = r2 * rinv;
                    float sn, cs;
                    __sincosf(P.pi_rca * r, &sn, &cs);
                    sm.d[p] = make_float4(d.x, d.y, d.z, r);
                    sm.fc[p] = 0.5f * cs + 0.5f;
                    if constexpr (BWD) {
                        sm.dfc[p] = -0.5f * P.pi_rca * sn;
                        sm.j[p] = j;
                    }
                }
            }
            na += __popc(m);
            if (na > kCapA) { // more in-cutoff angular neighbours than shared-memory slots
                if (lane == 0) atomicOr(&flags[0], NNP_FLAG_CAP_A);
                na = kCapA;
            }
        }
        if (na > na0) pm |= 1u << s;
    }
    if (lane == 0)
        for (int s = P.S; s <= NNP_MAX_SPECIES; ++s) sm.seg[s] = na;
    __syncwarp();
    *present = pm;
    return na;
}

// q-th pair of block (s,t): s != t -> (q / nt, q % nt); s == t -> q-th pair (a < b) of a triangle.
__device__ __forceinline__ void decode_pair(int q, bool same, int nt, float inv_nt, int &a, int &b)
{
    if (same) {
        int bb = (int)((1.0f + sqrtf(8.0f * (float)q + 1.0f)) * 0.5f);
        if (bb * (bb - 1) / 2 > q) --bb;
        if ((bb + 1) * bb / 2 <= q) ++bb;
        b = bb;
        a = q - bb * (bb - 1) / 2;
    } else {
        int aa = (int)(((float)q + 0.5f) * inv_nt);
        int rem = q - aa * nt;
        if (rem < 0) { --aa; rem += nt; }
        if (rem >= nt) { ++aa; rem -= nt; }
        a = aa;
        b = rem;
    }
}

__device__ __forceinline__ int pair_block(int S, int s, int t) { return s * (2 * S + 1 - s) / 2 + (t - s); }

__global__ void __launch_bounds__(kWarps * 32)
k_aev_forward(int n, AevParams P, const float4 *__restrict__ pos, const int *__restrict__ nbr_r,
              const uint16_t *__restrict__ seg_r, const int *__restrict__ nbr_a,
              const uint16_t *__restrict__ seg_a, float *__restrict__ G, int *__restrict__ flags)
{
    __shared__ WarpSmem smem[kWarps];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int i = blockIdx.x * kWarps + wid;
    if (i >= n) return;
    WarpSmem &sm = smem[wid];
    const float4 pi = pos[i];
    float *Grow = G + (size_t)i * P.kpad;

    // ---- radial block: G[s*16+k] = 1/4 sum_j exp(-eta_r (r-ShfR_k)^2) fc(r)
    {
        const uint16_t *sg = seg_r + (size_t)i * NNP_MAX_SPECIES; // sg[S..7] = row length (S <= 7)
        const int *row = nbr_r + (size_t)i * P.cap_r;
        for (int s = 0; s < P.S; ++s) {
            const int a_beg = sg[s], a_end = sg[s + 1];
            if (a_end == a_beg) {
                if (lane < NNP_NSHF_R) Grow[s * NNP_NSHF_R + lane] = 0.f;
                continue;
            }
            float acc[NNP_NSHF_R];
#pragma unroll
            for (int k = 0; k < NNP_NSHF_R; ++k) acc[k] = 0.f;
            for (int a = a_beg + lane; a < a_end; a += 32) {
                const float3 d = min_image(pi, pos[row[a]], P);
                const float r2 = d.x * d.x + d.y * d.y + d.z * d.z;
                if (r2 < P.rcr2) {
                    const float r = r2 * rsqrtf(r2);
                    const float fc = 0.125f * __cosf(P.pi_rcr * r) + 0.125f; // (1/4) fc
#pragma unroll
                    for (int k = 0; k < NNP_NSHF_R; ++k) {
                        const float u = r - P.shf_r[k];
                        acc[k] = fmaf(fc, ex2(P.neg_eta_r_log2e * u * u), acc[k]);
                    }
                }
            }
            butterfly_reduce<NNP_NSHF_R>(acc, lane);
            if ((lane & 1) == 0) Grow[s * NNP_NSHF_R + (lane >> 1)] = acc[0];
        }
        for (int q = P.aev_len + lane; q < P.kpad; q += 32) Grow[q] = 0.f; // zero padding columns
    }

    // ---- angular block
    unsigned present;
    stage_angular<false>(sm, P, i, lane, pi, pos, nbr_a, seg_a, flags, &present);
    unsigned done = 0; // bit p: block p written by the pair loop
    for (unsigned ms = present; ms; ms &= ms - 1) {
        const int s = __ffs(ms) - 1;
        const int a0 = sm.seg[s], ns = sm.seg[s + 1] - a0;
        for (unsigned mt = ms; mt; mt &= mt - 1) {
            const int t = __ffs(mt) - 1;
            const int b0 = sm.seg[t], nt = sm.seg[t + 1] - b0;
            const int npairs = (s == t) ? ns * (ns - 1) / 2 : ns * nt;
            if (npairs == 0) continue;
            const int p = pair_block(P.S, s, t);
            done |= 1u << p;
            const float inv_nt = 1.0f / (float)nt;
            float acc[NNP_ANG_BLOCK];
#pragma unroll
            for (int q = 0; q < NNP_ANG_BLOCK; ++q) acc[q] = 0.f;
            for (int q = lane; q < npairs; q += 32) {
                int ia, ib;
                decode_pair(q, s == t, nt, inv_nt, ia, ib);
                const float4 dj = sm.d[a0 + ia], dk = sm.d[b0 + ib];
                const float ff = 2.0f * sm.fc[a0 + ia] * sm.fc[b0 + ib];
                const float c = 0.95f * (dj.x * dk.x + dj.y * dk.y + dj.z * dk.z) * __frcp_rn(dj.w * dk.w);
                const float sn = sqrtf(fmaxf(1.0f - c * c, 0.f));
                const float rb = 0.5f * (dj.w + dk.w);
                float fz[NNP_NSHF_Z];
#pragma unroll
                for (int z = 0; z < NNP_NSHF_Z; ++z) {
                    const float base = fmaf(0.5f, c * P.cos_z[z] + sn * P.sin_z[z], 0.5f);
                    fz[z] = ex2(P.zeta * lg2(fmaxf(base, 0.f)));
                }
#pragma unroll
                for (int a = 0; a < NNP_NSHF_A; ++a) {
                    const float u = rb - P.shf_a[a];
                    const float ra = ff * ex2(P.neg_eta_a_log2e * u * u);
#pragma unroll
                    for (int z = 0; z < NNP_NSHF_Z; ++z) acc[a * NNP_NSHF_Z + z] = fmaf(ra, fz[z], acc[a * NNP_NSHF_Z + z]);
                }
            }
            butterfly_reduce<NNP_ANG_BLOCK>(acc, lane);
            Grow[P.n_rad + p * NNP_ANG_BLOCK + lane] = acc[0];
        }
    }
    const int nblocks = P.S * (P.S + 1) / 2;
    for (int p = 0; p < nblocks; ++p)
        if (!((done >> p) & 1u)) Grow[P.n_rad + p * NNP_ANG_BLOCK + lane] = 0.f;
}

// Reverse pass: g = dE/dG_i (row of dG, times inv_nets).  Adds -dE/dx to frc for the centre and its neighbours.
__global__ void __launch_bounds__(kWarps * 32)
k_aev_backward(int n, AevParams P, const float4 *__restrict__ pos, const int *__restrict__ nbr_r,
               const uint16_t *__restrict__ seg_r, const int *__restrict__ nbr_a,
               const uint16_t *__restrict__ seg_a, const float *__restrict__ dG, float inv_nets,
               float4 *__restrict__ frc, int *__restrict__ flags)
{
    extern __shared__ __align__(16) uint8_t smem_dyn[];
    WarpSmemBwd *smem = reinterpret_cast<WarpSmemBwd *>(smem_dyn);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int i = blockIdx.x * kWarps + wid;
    if (i >= n) return;
    WarpSmemBwd &sm = smem[wid];
    const float4 pi = pos[i];
    const float *grow = dG + (size_t)i * P.kpad;
    float fi[3] = {0.f, 0.f, 0.f}; // dE/dd summed over this lane's terms (force on i = +sum)

    // ---- radial: dE/dr_ij = sum_k g[s_j*16+k] * 1/4 e_k (-2 eta (r-ShfR_k) fc + fc')
    {
        const uint16_t *sg = seg_r + (size_t)i * NNP_MAX_SPECIES;
        const int *row = nbr_r + (size_t)i * P.cap_r;
        const float m2eta = -2.0f * P.eta_r;
        for (int s = 0; s < P.S; ++s) {
            const int a_beg = sg[s], a_end = sg[s + 1];
            if (a_end == a_beg) continue;
            float gr[NNP_NSHF_R];
            const float sc0 = 0.25f * inv_nets;
#pragma unroll
            for (int k4 = 0; k4 < NNP_NSHF_R / 4; ++k4) {
                const float4 v = *reinterpret_cast<const float4 *>(grow + s * NNP_NSHF_R + 4 * k4);
                gr[4 * k4] = v.x * sc0; gr[4 * k4 + 1] = v.y * sc0;
                gr[4 * k4 + 2] = v.z * sc0; gr[4 * k4 + 3] = v.w * sc0;
            }
            for (int a = a_beg + lane; a < a_end; a += 32) {
                const int j = row[a];
                const float3 d = min_image(pi, pos[j], P);
                const float r2 = d.x * d.x + d.y * d.y + d.z * d.z;
                if (r2 < P.rcr2) {
                    const float rinv = rsqrtf(r2);
                    const float r = r2 * rinv;
                    float sn, cs;
                    __sincosf(P.pi_rcr * r, &sn, &cs);
                    const float fc = 0.5f * cs + 0.5f;
                    const float dfc = -0.5f * P.pi_rcr * sn;
                    float dEdr = 0.f;
#pragma unroll
                    for (int k = 0; k < NNP_NSHF_R; ++k) {
                        const float u = r - P.shf_r[k];
                        const float e = ex2(P.neg_eta_r_log2e * u * u);
                        dEdr = fmaf(gr[k] * e, fmaf(m2eta * u, fc, dfc), dEdr);
                    }
                    const float sc = dEdr * rinv;
                    const float vx = sc * d.x, vy = sc * d.y, vz = sc * d.z;
                    atomicAdd(&frc[j], make_float4(-vx, -vy, -vz, 0.f));
                    fi[0] += vx; fi[1] += vy; fi[2] += vz;
                }
            }
        }
    }

    // ---- angular
    unsigned present;
    const int na = stage_angular<true>(sm, P, i, lane, pi, pos, nbr_a, seg_a, flags, &present);
    const bool arena = na * (na - 1) / 2 <= kArena; // warp-uniform
    if (!arena) {
        for (int a = lane; a < na; a += 32) { sm.f[a][0] = 0.f; sm.f[a][1] = 0.f; sm.f[a][2] = 0.f; }
        __syncwarp();
    }
    const float k_ang0 = 0.5f * P.zeta * 0.95f;
    const float m2eta_a = -2.0f * P.eta_a;
    for (unsigned ms = present; ms; ms &= ms - 1) {
        const int s = __ffs(ms) - 1;
        const int a0 = sm.seg[s], ns = sm.seg[s + 1] - a0;
        for (unsigned mt = ms; mt; mt &= mt - 1) {
            const int t = __ffs(mt) - 1;
            const int b0 = sm.seg[t], nt = sm.seg[t + 1] - b0;
            const int npairs = (s == t) ? ns * (ns - 1) / 2 : ns * nt;
            if (npairs == 0) continue;
            const int p = pair_block(P.S, s, t);
            const float inv_nt = 1.0f / (float)nt;
            float gw[NNP_ANG_BLOCK];
            const float *gp = grow + P.n_rad + p * NNP_ANG_BLOCK;
            const float sc0 = 2.0f * inv_nets; // the prefactor 2 of the angular term
#pragma unroll
            for (int q4 = 0; q4 < NNP_ANG_BLOCK / 4; ++q4) {
                const float4 v = *reinterpret_cast<const float4 *>(gp + 4 * q4);
                gw[4 * q4] = v.x * sc0; gw[4 * q4 + 1] = v.y * sc0;
                gw[4 * q4 + 2] = v.z * sc0; gw[4 * q4 + 3] = v.w * sc0;
            }
            for (int q = lane; q < npairs; q += 32) {
                int ia, ib;
                decode_pair(q, s == t, nt, inv_nt, ia, ib);
                ia += a0; ib += b0;
                const float4 dj = sm.d[ia], dk = sm.d[ib];
                const float fj = sm.fc[ia], fk = sm.fc[ib];
                const float rj_inv = __frcp_rn(dj.w), rk_inv = __frcp_rn(dk.w);
                const float rjk_inv = rj_inv * rk_inv;
                const float cs = (dj.x * dk.x + dj.y * dk.y + dj.z * dk.z) * rjk_inv; // cos(theta)
                const float c = 0.95f * cs;
                const float sn = sqrtf(fmaxf(1.0f - c * c, 0.f));
                const float rb = 0.5f * (dj.w + dk.w);
                float fz[NNP_NSHF_Z], dfz[NNP_NSHF_Z]; // F_z and dF_z/dcos(theta)
                const float k_ang = k_ang0 * __frcp_rn(sn);
#pragma unroll
                for (int z = 0; z < NNP_NSHF_Z; ++z) {
                    const float base = fmaxf(fmaf(0.5f, c * P.cos_z[z] + sn * P.sin_z[z], 0.5f), 0.f);
                    const float pw = ex2((P.zeta - 1.0f) * lg2(base)); // base^(zeta-1)
                    fz[z] = pw * base;
                    // dF/dtheta' = -(zeta/2) sin(theta'-phi) base^(zeta-1); dtheta'/dcos = -0.95/sn
                    dfz[z] = k_ang * (sn * P.cos_z[z] - c * P.sin_z[z]) * pw;
                }
                float Az[NNP_NSHF_Z] = {0.f, 0.f, 0.f, 0.f};
                float dE_drb = 0.f;
#pragma unroll
                for (int a = 0; a < NNP_NSHF_A; ++a) {
                    const float u = rb - P.shf_a[a];
                    const float ra = ex2(P.neg_eta_a_log2e * u * u);
                    float Ba = 0.f;
#pragma unroll
                    for (int z = 0; z < NNP_NSHF_Z; ++z) {
                        const float w = gw[a * NNP_NSHF_Z + z];
                        Az[z] = fmaf(w, ra, Az[z]);
                        Ba = fmaf(w, fz[z], Ba);
                    }
                    dE_drb = fmaf(Ba * ra, m2eta_a * u, dE_drb);
                }
                float T = 0.f, dE_dcs = 0.f;
#pragma unroll
                for (int z = 0; z < NNP_NSHF_Z; ++z) {
                    T = fmaf(Az[z], fz[z], T);
                    dE_dcs = fmaf(Az[z], dfz[z], dE_dcs);
                }
                const float ff = fj * fk;
                dE_dcs *= ff;
                const float half_drb = 0.5f * dE_drb * ff;
                const float dE_drj = fmaf(T * sm.dfc[ia], fk, half_drb);
                const float dE_drk = fmaf(T * fj, sm.dfc[ib], half_drb);
                const float beta = dE_dcs * rjk_inv;
                const float alj = (dE_drj - dE_dcs * cs * rj_inv) * rj_inv;
                const float alk = (dE_drk - dE_dcs * cs * rk_inv) * rk_inv;
                if (arena) {
                    const int slot = ib * (ib - 1) / 2 + ia; // ia < ib
                    sm.alo[slot] = alj; sm.ahi[slot] = alk; sm.bet[slot] = beta;
                } else {
                    atomicAdd(&sm.f[ia][0], alj * dj.x + beta * dk.x);
                    atomicAdd(&sm.f[ia][1], alj * dj.y + beta * dk.y);
                    atomicAdd(&sm.f[ia][2], alj * dj.z + beta * dk.z);
                    atomicAdd(&sm.f[ib][0], beta * dj.x + alk * dk.x);
                    atomicAdd(&sm.f[ib][1], beta * dj.y + alk * dk.y);
                    atomicAdd(&sm.f[ib][2], beta * dj.z + alk * dk.z);
                }
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
            for (int b = 0; b < a; ++b) {
                const int slot = a * (a - 1) / 2 + b;
                const float be = sm.bet[slot];
                const float4 db = sm.d[b];
                asum += sm.ahi[slot];
                fx = fmaf(be, db.x, fx); fy = fmaf(be, db.y, fy); fz = fmaf(be, db.z, fz);
            }
            for (int b = a + 1; b < na; ++b) {
                const int slot = b * (b - 1) / 2 + a;
                const float be = sm.bet[slot];
                const float4 db = sm.d[b];
                asum += sm.alo[slot];
                fx = fmaf(be, db.x, fx); fy = fmaf(be, db.y, fy); fz = fmaf(be, db.z, fz);
            }
            fx = fmaf(asum, da.x, fx); fy = fmaf(asum, da.y, fy); fz = fmaf(asum, da.z, fz);
        } else {
            fx = sm.f[a][0]; fy = sm.f[a][1]; fz = sm.f[a][2];
        }
        atomicAdd(&frc[sm.j[a]], make_float4(-fx, -fy, -fz, 0.f));
        fi[0] += fx; fi[1] += fy; fi[2] += fz;
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) fi[c] += __shfl_xor_sync(0xffffffffu, fi[c], o);
    }
    if (lane == 0) atomicAdd(&frc[i], make_float4(fi[0], fi[1], fi[2], 0.f));
}

} // namespace

void nnp_launch_aev_forward(nnp_ctx *c)
{
    k_aev_forward<<<nnp_div_up(c->n, kWarps), kWarps * 32, 0, c->stream>>>(c->n, c->aev, c->pos, c->nbr_r, c->seg_r,
                                                                         c->nbr_a, c->seg_a, c->G, c->flags);
    c->launches += 1;
}

void nnp_launch_aev_backward(nnp_ctx *c, float inv_nets)
{
    static bool attr_set = false;
    const int smem = (int)sizeof(WarpSmemBwd) * kWarps;
    if (!attr_set) {
        cudaFuncSetAttribute(k_aev_backward, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        attr_set = true;
    }
    k_aev_backward<<<nnp_div_up(c->n, kWarps), kWarps * 32, smem, c->stream>>>(
        c->n, c->aev, c->pos, c->nbr_r, c->seg_r, c->nbr_a, c->seg_a, c->dG, inv_nets, c->frc, c->flags);
    c->launches += 1;
}
