// Stage 2 (AEV forward) and the AEV half of stage 4 (reverse pass + force scatter).
// Definition: SURVEY.md 8(c) O2/O3/O6 (PAPER.md L61 cosine switch, L79 Gaussian radial basis, L443 angular form
// (0.5+0.5cos(theta-theta_n))^zeta, L55 pairs of edges with a common centre, L65/L176 forces by reverse mode).
//
// One warp per centre atom.  Neighbour rows are grouped by neighbour species (stage 1), so
//   radial:  lane = neighbour, 16 Gaussians in registers per species segment, butterfly reduction over lanes;
//   angular: the in-cutoff neighbours are compacted into shared memory (dx,dy,dz,r | fc | fc'), then for each
//            species pair (s,t) lanes take pairs (j,k), keep the 8x4 terms in 32 registers and a 31-shuffle
//            butterfly leaves feature `lane` of that 32-wide block in lane `lane` -> one coalesced 128 B store.
// Triplets are enumerated on the fly and never stored (the paper's GraphAngularExtension stores them, L55).
// cos(theta' - ShfZ) with theta' = acos(0.95 cos theta) is expanded as c' cos ShfZ + sqrt(1-c'^2) sin ShfZ: no acos.
#include "nnp_internal.cuh"

namespace {

constexpr int kWarps = 4;
constexpr int kCapA = 64; // shared-memory slots for in-cutoff angular neighbours per centre

struct WarpSmem {
    float4 d[kCapA];   // dx, dy, dz, r
    float fc[kCapA];
    float dfc[kCapA];  // backward only
    float f[kCapA][3]; // backward: dE/dd accumulators per neighbour
    int j[kCapA];
    int seg[NNP_MAX_SPECIES + 1];
};

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

__device__ __forceinline__ void load_seg(const uint16_t *seg, int (&out)[NNP_MAX_SPECIES + 1])
{
    const uint4 u = *reinterpret_cast<const uint4 *>(seg);
    out[0] = u.x & 0xffff; out[1] = u.x >> 16; out[2] = u.y & 0xffff; out[3] = u.y >> 16;
    out[4] = u.z & 0xffff; out[5] = u.z >> 16; out[6] = u.w & 0xffff; out[7] = u.w >> 16;
    out[8] = out[7];
}

// Compacts the angular neighbours with r < rca into shared memory, keeping the species grouping.
template <bool BWD>
__device__ __forceinline__ int stage_angular(WarpSmem &sm, const AevParams &P, int i, int lane, const float4 pi,
                                             const float4 *__restrict__ pos, const int *__restrict__ nbr_a,
                                             const uint16_t *__restrict__ seg_a, int *__restrict__ flags)
{
    int sg[NNP_MAX_SPECIES + 1];
    load_seg(seg_a + (size_t)i * NNP_MAX_SPECIES, sg);
    const int *row = nbr_a + (size_t)i * P.cap_a;
    const unsigned lt = (1u << lane) - 1u;
    int na = 0;
#pragma unroll
    for (int s = 0; s < NNP_MAX_SPECIES; ++s) {
        if (lane == 0) sm.seg[s] = na;
        if (s < P.S) {
            for (int a0 = sg[s]; a0 < sg[s + 1]; a0 += 32) {
                const int a = a0 + lane;
                bool hit = false;
                float3 d = make_float3(0.f, 0.f, 0.f);
                float r2 = 0.f;
                int j = 0;
                if (a < sg[s + 1]) {
                    j = row[a];
                    d = min_image(pi, pos[j], P);
                    r2 = d.x * d.x + d.y * d.y + d.z * d.z;
                    hit = r2 < P.rca2;
                }
                const unsigned m = __ballot_sync(0xffffffffu, hit);
                if (hit) {
                    const int p = na + __popc(m & lt);
                    if (p < kCapA) {
                        const float r = sqrtf(r2);
                        float sn, cs;
                        __sincosf(P.pi_rca * r, &sn, &cs);
                        sm.d[p] = make_float4(d.x, d.y, d.z, r);
                        sm.fc[p] = 0.5f * cs + 0.5f;
                        if (BWD) {
                            sm.dfc[p] = -0.5f * P.pi_rca * sn;
                            sm.j[p] = j;
                            sm.f[p][0] = 0.f; sm.f[p][1] = 0.f; sm.f[p][2] = 0.f;
                        }
                    }
                }
                na += __popc(m);
                if (na > kCapA) { // more in-cutoff angular neighbours than shared-memory slots
                    if (lane == 0) atomicOr(&flags[0], NNP_FLAG_CAP_A);
                    na = kCapA;
                }
            }
        }
    }
    if (lane == 0) sm.seg[NNP_MAX_SPECIES] = na;
    __syncwarp();
    return na;
}

// q-th pair of block (s,t): s != t -> (q / nt, q % nt); s == t -> q-th pair (a < b) of a triangle.
__device__ __forceinline__ void decode_pair(int q, bool same, int nt, int &a, int &b)
{
    if (same) {
        // b = floor((1 + sqrt(8q+1)) / 2), a = q - b(b-1)/2, with an integer fix-up
        int bb = (int)((1.0f + sqrtf(8.0f * (float)q + 1.0f)) * 0.5f);
        while (bb * (bb - 1) / 2 > q) --bb;
        while ((bb + 1) * bb / 2 <= q) ++bb;
        b = bb;
        a = q - bb * (bb - 1) / 2;
    } else {
        a = q / nt;
        b = q - a * nt;
    }
}

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
            float acc[NNP_NSHF_R];
#pragma unroll
            for (int k = 0; k < NNP_NSHF_R; ++k) acc[k] = 0.f;
            const int a_beg = sg[s], a_end = sg[s + 1];
            for (int a = a_beg + lane; a < a_end; a += 32) {
                const float3 d = min_image(pi, pos[row[a]], P);
                const float r2 = d.x * d.x + d.y * d.y + d.z * d.z;
                if (r2 < P.rcr2) {
                    const float r = sqrtf(r2);
                    const float fc = 0.125f * __cosf(P.pi_rcr * r) + 0.125f; // (1/4) fc
#pragma unroll
                    for (int k = 0; k < NNP_NSHF_R; ++k) {
                        const float u = r - P.shf_r[k];
                        acc[k] = fmaf(fc, exp2f(P.neg_eta_r_log2e * u * u), acc[k]);
                    }
                }
            }
            if (a_end > a_beg) butterfly_reduce<NNP_NSHF_R>(acc, lane);
            if ((lane & 1) == 0) Grow[s * NNP_NSHF_R + (lane >> 1)] = acc[0];
        }
        // zero padding columns aev_len..kpad
        for (int q = P.aev_len + lane; q < P.kpad; q += 32) Grow[q] = 0.f;
    }

    // ---- angular block
    stage_angular<false>(sm, P, i, lane, pi, pos, nbr_a, seg_a, flags);
    int p = 0;
    for (int s = 0; s < P.S; ++s) {
        const int a0 = sm.seg[s], ns = sm.seg[s + 1] - a0;
        for (int t = s; t < P.S; ++t, ++p) {
            const int b0 = sm.seg[t], nt = sm.seg[t + 1] - b0;
            const int npairs = (s == t) ? ns * (ns - 1) / 2 : ns * nt;
            float *out = Grow + P.n_rad + p * NNP_ANG_BLOCK;
            if (npairs == 0) { out[lane] = 0.f; continue; }
            float acc[NNP_ANG_BLOCK];
#pragma unroll
            for (int q = 0; q < NNP_ANG_BLOCK; ++q) acc[q] = 0.f;
            for (int q = lane; q < npairs; q += 32) {
                int ia, ib;
                decode_pair(q, s == t, nt, ia, ib);
                const float4 dj = sm.d[a0 + ia], dk = sm.d[b0 + ib];
                const float ff = 2.0f * sm.fc[a0 + ia] * sm.fc[b0 + ib];
                const float c = 0.95f * (dj.x * dk.x + dj.y * dk.y + dj.z * dk.z) * __frcp_rn(dj.w * dk.w);
                const float sn = sqrtf(fmaxf(1.0f - c * c, 0.f));
                const float rb = 0.5f * (dj.w + dk.w);
                float fz[NNP_NSHF_Z];
#pragma unroll
                for (int z = 0; z < NNP_NSHF_Z; ++z) {
                    const float base = 0.5f + 0.5f * (c * P.cos_z[z] + sn * P.sin_z[z]);
                    fz[z] = exp2f(P.zeta * __log2f(fmaxf(base, 0.f)));
                }
#pragma unroll
                for (int a = 0; a < NNP_NSHF_A; ++a) {
                    const float u = rb - P.shf_a[a];
                    const float ra = ff * exp2f(P.neg_eta_a_log2e * u * u);
#pragma unroll
                    for (int z = 0; z < NNP_NSHF_Z; ++z) acc[a * NNP_NSHF_Z + z] = fmaf(ra, fz[z], acc[a * NNP_NSHF_Z + z]);
                }
            }
            butterfly_reduce<NNP_ANG_BLOCK>(acc, lane);
            out[lane] = acc[0];
        }
    }
}

// Reverse pass: g = dE/dG_i (row of dG, times inv_nets).  Adds -dE/dx to frc for the centre and its neighbours.
__global__ void __launch_bounds__(kWarps * 32)
k_aev_backward(int n, AevParams P, const float4 *__restrict__ pos, const int *__restrict__ nbr_r,
               const uint16_t *__restrict__ seg_r, const int *__restrict__ nbr_a,
               const uint16_t *__restrict__ seg_a, const float *__restrict__ dG, float inv_nets,
               float4 *__restrict__ frc, int *__restrict__ flags)
{
    __shared__ WarpSmem smem[kWarps];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int i = blockIdx.x * kWarps + wid;
    if (i >= n) return;
    WarpSmem &sm = smem[wid];
    const float4 pi = pos[i];
    const float *grow = dG + (size_t)i * P.kpad;
    float fi[3] = {0.f, 0.f, 0.f}; // dE/dd summed over this lane's terms (force on i = +sum)

    // ---- radial: dE/dr_ij = sum_k g[s_j*16+k] * 1/4 e_k (-2 eta (r-ShfR_k) fc + fc')
    {
        const uint16_t *sg = seg_r + (size_t)i * NNP_MAX_SPECIES;
        const int *row = nbr_r + (size_t)i * P.cap_r;
        for (int s = 0; s < P.S; ++s) {
            const int a_beg = sg[s], a_end = sg[s + 1];
            if (a_end == a_beg) continue;
            float gr[NNP_NSHF_R];
#pragma unroll
            for (int k4 = 0; k4 < NNP_NSHF_R / 4; ++k4) {
                const float4 v = *reinterpret_cast<const float4 *>(grow + s * NNP_NSHF_R + 4 * k4);
                gr[4 * k4] = v.x * inv_nets; gr[4 * k4 + 1] = v.y * inv_nets;
                gr[4 * k4 + 2] = v.z * inv_nets; gr[4 * k4 + 3] = v.w * inv_nets;
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
                        const float e = exp2f(P.neg_eta_r_log2e * u * u);
                        dEdr = fmaf(gr[k] * e, fmaf(-2.0f * P.eta_r * u, fc, dfc), dEdr);
                    }
                    const float sc = 0.25f * dEdr * rinv;
                    const float vx = sc * d.x, vy = sc * d.y, vz = sc * d.z;
                    atomicAdd(&frc[j].x, -vx);
                    atomicAdd(&frc[j].y, -vy);
                    atomicAdd(&frc[j].z, -vz);
                    fi[0] += vx; fi[1] += vy; fi[2] += vz;
                }
            }
        }
    }

    // ---- angular
    const int na = stage_angular<true>(sm, P, i, lane, pi, pos, nbr_a, seg_a, flags);
    int p = 0;
    for (int s = 0; s < P.S; ++s) {
        const int a0 = sm.seg[s], ns = sm.seg[s + 1] - a0;
        for (int t = s; t < P.S; ++t, ++p) {
            const int b0 = sm.seg[t], nt = sm.seg[t + 1] - b0;
            const int npairs = (s == t) ? ns * (ns - 1) / 2 : ns * nt;
            if (npairs == 0) continue;
            float gw[NNP_ANG_BLOCK];
            const float *gp = grow + P.n_rad + p * NNP_ANG_BLOCK;
#pragma unroll
            for (int q4 = 0; q4 < NNP_ANG_BLOCK / 4; ++q4) {
                const float4 v = *reinterpret_cast<const float4 *>(gp + 4 * q4);
                gw[4 * q4] = v.x * inv_nets; gw[4 * q4 + 1] = v.y * inv_nets;
                gw[4 * q4 + 2] = v.z * inv_nets; gw[4 * q4 + 3] = v.w * inv_nets;
            }
            for (int q = lane; q < npairs; q += 32) {
                int ia, ib;
                decode_pair(q, s == t, nt, ia, ib);
                ia += a0; ib += b0;
                const float4 dj = sm.d[ia], dk = sm.d[ib];
                const float fj = sm.fc[ia], fk = sm.fc[ib];
                const float rjk_inv = __frcp_rn(dj.w * dk.w);
                const float cs = (dj.x * dk.x + dj.y * dk.y + dj.z * dk.z) * rjk_inv; // cos(theta)
                const float c = 0.95f * cs;
                const float sn = sqrtf(fmaxf(1.0f - c * c, 0.f));
                const float rb = 0.5f * (dj.w + dk.w);
                float fz[NNP_NSHF_Z], dfz[NNP_NSHF_Z]; // F_z and dF_z/dcos(theta)
                const float k_ang = 0.5f * P.zeta * 0.95f * __frcp_rn(sn);
#pragma unroll
                for (int z = 0; z < NNP_NSHF_Z; ++z) {
                    const float base = fmaxf(0.5f + 0.5f * (c * P.cos_z[z] + sn * P.sin_z[z]), 0.f);
                    const float pw = exp2f((P.zeta - 1.0f) * __log2f(base)); // base^(zeta-1)
                    fz[z] = pw * base;
                    // dF/dtheta' = -(zeta/2) sin(theta'-phi) base^(zeta-1); dtheta'/dcos = -0.95/sn
                    dfz[z] = k_ang * (sn * P.cos_z[z] - c * P.sin_z[z]) * pw;
                }
                float Az[NNP_NSHF_Z] = {0.f, 0.f, 0.f, 0.f};
                float dE_drb = 0.f;
#pragma unroll
                for (int a = 0; a < NNP_NSHF_A; ++a) {
                    const float u = rb - P.shf_a[a];
                    const float ra = exp2f(P.neg_eta_a_log2e * u * u);
                    float Ba = 0.f;
#pragma unroll
                    for (int z = 0; z < NNP_NSHF_Z; ++z) {
                        const float w = gw[a * NNP_NSHF_Z + z];
                        Az[z] = fmaf(w, ra, Az[z]);
                        Ba = fmaf(w, fz[z], Ba);
                    }
                    dE_drb = fmaf(Ba * ra, -2.0f * P.eta_a * u, dE_drb);
                }
                float T = 0.f, dE_dcs = 0.f;
#pragma unroll
                for (int z = 0; z < NNP_NSHF_Z; ++z) {
                    T = fmaf(Az[z], fz[z], T);
                    dE_dcs = fmaf(Az[z], dfz[z], dE_dcs);
                }
                const float ff = 2.0f * fj * fk;
                dE_dcs *= ff;
                dE_drb *= ff;
                const float dE_drj = 0.5f * dE_drb + 2.0f * T * sm.dfc[ia] * fk;
                const float dE_drk = 0.5f * dE_drb + 2.0f * T * fj * sm.dfc[ib];
                const float rj_inv = __frcp_rn(dj.w), rk_inv = __frcp_rn(dk.w);
                const float beta = dE_dcs * rjk_inv;
                const float alj = (dE_drj - dE_dcs * cs * rj_inv) * rj_inv;
                const float alk = (dE_drk - dE_dcs * cs * rk_inv) * rk_inv;
                const float vjx = alj * dj.x + beta * dk.x, vjy = alj * dj.y + beta * dk.y, vjz = alj * dj.z + beta * dk.z;
                const float vkx = beta * dj.x + alk * dk.x, vky = beta * dj.y + alk * dk.y, vkz = beta * dj.z + alk * dk.z;
                atomicAdd(&sm.f[ia][0], vjx); atomicAdd(&sm.f[ia][1], vjy); atomicAdd(&sm.f[ia][2], vjz);
                atomicAdd(&sm.f[ib][0], vkx); atomicAdd(&sm.f[ib][1], vky); atomicAdd(&sm.f[ib][2], vkz);
                fi[0] += vjx + vkx; fi[1] += vjy + vky; fi[2] += vjz + vkz;
            }
        }
    }
    __syncwarp();
    for (int a = lane; a < na; a += 32) {
        const int j = sm.j[a];
        atomicAdd(&frc[j].x, -sm.f[a][0]);
        atomicAdd(&frc[j].y, -sm.f[a][1]);
        atomicAdd(&frc[j].z, -sm.f[a][2]);
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) fi[c] += __shfl_xor_sync(0xffffffffu, fi[c], o);
    }
    if (lane == 0) {
        atomicAdd(&frc[i].x, fi[0]);
        atomicAdd(&frc[i].y, fi[1]);
        atomicAdd(&frc[i].z, fi[2]);
    }
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
    k_aev_backward<<<nnp_div_up(c->n, kWarps), kWarps * 32, 0, c->stream>>>(
        c->n, c->aev, c->pos, c->nbr_r, c->seg_r, c->nbr_a, c->seg_a, c->dG, inv_nets, c->frc, c->flags);
    c->launches += 1;
}
