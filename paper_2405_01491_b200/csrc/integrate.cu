// Stage 5: velocity Verlet with the Verlet-skin rebuild test on the device (fennol_md NVE, PAPER.md L307;
// skin and rebuild policy L341, reading C2), the per-structure energy sum (L176, reading B5) and the
// permutations between the caller's atom order and the internal (species, cell) order.
#include "nnp_internal.cuh"

namespace {

constexpr int T = 256;

// v += dt/2 a(F); x += dt v; request a list rebuild iff |x - xref|^2 > (skin/2)^2 for any atom.
__global__ void k_kick_drift(int n, float4 *__restrict__ pos, float4 *__restrict__ vel, const float4 *__restrict__ frc,
                             const float4 *__restrict__ xref, const int *__restrict__ spc,
                             const float *__restrict__ inv_mass_conv, float dt, float half_skin2, int *__restrict__ flags)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    bool moved = false;
    if (i < n) {
        const float k = 0.5f * dt * inv_mass_conv[spc[i]];
        float4 v = vel[i], x = pos[i];
        const float4 f = frc[i], r = xref[i];
        v.x = fmaf(k, f.x, v.x); v.y = fmaf(k, f.y, v.y); v.z = fmaf(k, f.z, v.z);
        x.x = fmaf(dt, v.x, x.x); x.y = fmaf(dt, v.y, x.y); x.z = fmaf(dt, v.z, x.z);
        vel[i] = v;
        pos[i] = x;
        const float dx = x.x - r.x, dy = x.y - r.y, dz = x.z - r.z;
        moved = dx * dx + dy * dy + dz * dz > half_skin2;
    }
    if (__syncthreads_or(moved) && threadIdx.x == 0) flags[1] = 1;
}

// Philox4x32-10 (Salmon et al., SC'11): counter (atom, step, 0, 0), key = seed.
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1,
                                              uint32_t (&out)[4])
{
#pragma unroll
    for (int round = 0; round < 10; ++round) {
        if (round) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
        const uint32_t h0 = __umulhi(0xD2511F53u, c0), l0 = 0xD2511F53u * c0;
        const uint32_t h1 = __umulhi(0xCD9E8D57u, c2), l1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = h1 ^ c1 ^ k0, n2 = h0 ^ c3 ^ k1;
        c0 = n0; c1 = l1; c2 = n2; c3 = l0;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Langevin dynamics, BAOAB ("Langevin dynamics (using the BAOAB scheme)", L323):
// B: v += dt/2 a(F); A: x += dt/2 v; O: v = c1 v + c2[species] xi; A: x += dt/2 v; then the rebuild test.
// xi: three standard normals per atom and step, keyed by the ORIGINAL atom index and the device-side step counter
// flags[4] (so the numbers do not depend on the internal atom order or on how many steps one call enqueues):
// u = ((r >> 9) + 1/2) 2^-23 (exact in fp32), Box-Muller.  gamma = 0 never comes here (velocity Verlet kernel above).
__global__ void k_kick_drift_langevin(int n, float4 *__restrict__ pos, float4 *__restrict__ vel, const float4 *__restrict__ frc,
                                      const float4 *__restrict__ xref, const int *__restrict__ spc, const int *__restrict__ orig,
                                      const float *__restrict__ inv_mass_conv, const float *__restrict__ c2_s, float c1, float dt,
                                      float half_skin2, uint32_t seed_lo, uint32_t seed_hi, int *__restrict__ flags, int n_user)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    bool moved = false;
    if (i < n) {
        const int s = spc[i];
        const float k = 0.5f * dt * inv_mass_conv[s], hdt = 0.5f * dt, c2 = c2_s[s];
        float4 v = vel[i], x = pos[i];
        const float4 f = frc[i], r = xref[i];
        v.x = fmaf(k, f.x, v.x); v.y = fmaf(k, f.y, v.y); v.z = fmaf(k, f.z, v.z);
        x.x = fmaf(hdt, v.x, x.x); x.y = fmaf(hdt, v.y, x.y); x.z = fmaf(hdt, v.z, x.z);
        uint32_t rn[4];
        philox4x32_10((uint32_t)(orig[i] % n_user), (uint32_t)flags[4], 0u, 0u, seed_lo, seed_hi, rn); // (copies of a small cell: the atom's noise)
        float u[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) u[q] = ((float)(rn[q] >> 9) + 0.5f) * 1.1920928955078125e-07f; // 2^-23
        const float a = sqrtf(-2.0f * logf(u[0])), b = sqrtf(-2.0f * logf(u[2]));
        float sn, cs, cs2;
        sincospif(2.0f * u[1], &sn, &cs);
        cs2 = cospif(2.0f * u[3]);
        v.x = fmaf(c1, v.x, c2 * (a * cs)); v.y = fmaf(c1, v.y, c2 * (a * sn)); v.z = fmaf(c1, v.z, c2 * (b * cs2));
        x.x = fmaf(hdt, v.x, x.x); x.y = fmaf(hdt, v.y, x.y); x.z = fmaf(hdt, v.z, x.z);
        vel[i] = v;
        pos[i] = x;
        const float dx = x.x - r.x, dy = x.y - r.y, dz = x.z - r.z;
        moved = dx * dx + dy * dy + dz * dz > half_skin2;
    }
    if (__syncthreads_or(moved) && threadIdx.x == 0) flags[1] = 1;
}

// out[m] += v for the lanes with ok; the lanes of a warp that share a structure add once (the internal order keeps the
// atoms of a structure together inside a species bucket, so a warp meets one or two structures)
__device__ __forceinline__ void add_per_structure(bool ok, int m, double v, double *__restrict__ out)
{
    const unsigned peers = __match_any_sync(0xffffffffu, ok ? m : -1);
    const int lane = threadIdx.x & 31;
    const int leader = __ffs(peers) - 1;
    double s = 0.0;
    for (unsigned rest = peers; rest; rest &= rest - 1) s += __shfl_sync(peers, v, __ffs(rest) - 1);
    if (ok && lane == leader) atomicAdd(&out[m], s);
}

// v += dt/2 a(F); kinetic energy sum_i m v^2 / (2 accel_conv) accumulated in fp64.
__global__ void k_kick_ke(int n, float4 *__restrict__ vel, const float4 *__restrict__ frc, const int *__restrict__ spc,
                          const float *__restrict__ inv_mass_conv, const float *__restrict__ mass, float dt,
                          float inv_accel_conv, float inv_rep, const int *__restrict__ mol, int single, double *__restrict__ ekin,
                          int *__restrict__ step_ctr)
{
    if (step_ctr && blockIdx.x == 0 && threadIdx.x == 0) *step_ctr += 1; // Langevin step counter (read by the next drift kernel)
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    float ke = 0.f;
    if (i < n) {
        const int s = spc[i];
        const float k = 0.5f * dt * inv_mass_conv[s];
        float4 v = vel[i];
        const float4 f = frc[i];
        v.x = fmaf(k, f.x, v.x); v.y = fmaf(k, f.y, v.y); v.z = fmaf(k, f.z, v.z);
        vel[i] = v;
        ke = 0.5f * mass[s] * (v.x * v.x + v.y * v.y + v.z * v.z) * inv_accel_conv * inv_rep;
    }
    if (!single) { // one kinetic energy per structure (replica batches)
        add_per_structure(i < n, i < n ? mol[i] : -1, (double)ke, ekin);
        return;
    }
    __shared__ double part[T / 32];
    double d = (double)ke;
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) d += __shfl_xor_sync(0xffffffffu, d, o);
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = d;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int w = 0; w < T / 32; ++w) s += part[w];
        atomicAdd(ekin, s);
    }
}

// E_mol += e_atom * inv_nets + e_shift[species]   (fp64 accumulation; block-reduced when there is one structure)
__global__ void k_energy_reduce(int n, const float *__restrict__ e_atom, const int *__restrict__ spc,
                                const int *__restrict__ mol, const float *__restrict__ e_shift, float inv_nets,
                                double inv_rep, int single, double *__restrict__ e_mol)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    double e = 0.0;
    if (i < n) e = ((double)e_atom[i] * (double)inv_nets + (double)e_shift[spc[i]]) * inv_rep; // per cell of a replicated small cell
    if (!single) {
        add_per_structure(i < n, i < n ? mol[i] : -1, e, e_mol);
        return;
    }
    __shared__ double part[T / 32];
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = e;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int w = 0; w < T / 32; ++w) s += part[w];
        atomicAdd(&e_mol[0], s);
    }
}

// (n_user: the caller's atoms; internal atoms with orig >= n_user are the extra copies of a replicated small cell)
__global__ void k_unpermute3(int n, const float4 *__restrict__ src, const int *__restrict__ orig, int n_user, float *__restrict__ dst)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float4 v = src[i];
    const int o = orig[i];
    if (o >= n_user) return;
    dst[3 * o] = v.x; dst[3 * o + 1] = v.y; dst[3 * o + 2] = v.z;
}

__global__ void k_permute_in3(int n, const float *__restrict__ src, const int *__restrict__ orig, int n_user, float4 *__restrict__ dst)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int o = orig[i] % n_user; // (the copies of a replicated small cell take their atom's value)
    dst[i] = make_float4(src[3 * o], src[3 * o + 1], src[3 * o + 2], 0.f);
}

__global__ void k_unpermute3x2(int n, const float4 *__restrict__ srcA, const float4 *__restrict__ srcB,
                               const int *__restrict__ orig, int n_user, float *__restrict__ dstA, float *__restrict__ dstB)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float4 a = srcA[i], b = srcB[i];
    const int o = orig[i];
    if (o >= n_user) return;
    dstA[3 * o] = a.x; dstA[3 * o + 1] = a.y; dstA[3 * o + 2] = a.z;
    dstB[3 * o] = b.x; dstB[3 * o + 1] = b.y; dstB[3 * o + 2] = b.z;
}

__global__ void k_permute_in3x2(int n, const float *__restrict__ srcA, const float *__restrict__ srcB,
                                const int *__restrict__ orig, int n_user, float4 *__restrict__ dstA, float4 *__restrict__ dstB)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int o = orig[i] % n_user;
    dstA[i] = make_float4(srcA[3 * o], srcA[3 * o + 1], srcA[3 * o + 2], 0.f);
    dstB[i] = make_float4(srcB[3 * o], srcB[3 * o + 1], srcB[3 * o + 2], 0.f);
}

__global__ void k_pack_result(const double *__restrict__ e_mol, const double *__restrict__ ekin,
                              const int *__restrict__ flags, double *__restrict__ res)
{
    if (threadIdx.x == 0) {
        res[0] = e_mol[0]; res[1] = ekin[0];
        res[2] = (double)flags[0]; res[3] = (double)flags[1]; res[4] = (double)flags[2];
    }
}

// Replicated small cell (nnp_set_system_cell): the copies are kept bit-identical to copy 0 - a copy's position is its atom's
// plus the copy's lattice shift, its velocity and force are its atom's.  (Left alone the copies drift apart by the rounding
// of x + shift + dt v and by the summation order of the force scatter, and the supercell stops being periodic in the cell.)
__global__ void k_stage_copy0(int n, const int *__restrict__ orig, int n_user, const float4 *__restrict__ a, const float4 *__restrict__ b,
                              float4 *__restrict__ stage)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int e = orig[i];
    if (e >= n_user) return;
    stage[e] = a[i];
    if (b) stage[n_user + e] = b[i];
}

struct RepCell { float cu[9]; };
__global__ void k_spread_copy0(int n, const int *__restrict__ orig, int n_user, int m0, int m1, RepCell rc,
                               const float4 *__restrict__ stage, float4 *__restrict__ a, float4 *__restrict__ b, int shift_a)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int e = orig[i];
    if (e < n_user) return;
    const int at = e % n_user, copy = e / n_user;
    float4 v = stage[at];
    if (shift_a) {
        const float k0 = (float)(copy % m0), k1 = (float)((copy / m0) % m1), k2 = (float)(copy / (m0 * m1));
        v.x += k0 * rc.cu[0] + k1 * rc.cu[3] + k2 * rc.cu[6];
        v.y += k0 * rc.cu[1] + k1 * rc.cu[4] + k2 * rc.cu[7];
        v.z += k0 * rc.cu[2] + k1 * rc.cu[5] + k2 * rc.cu[8];
    }
    a[i] = v;
    if (b) b[i] = stage[n_user + at];
}

} // namespace

int nnp_launch_sync_copies(nnp_ctx *c, int what)
{
    if (c->rep <= 1) return NNP_OK;
    const int nb = nnp_div_up(c->n, T);
    RepCell rcell;
    for (int q = 0; q < 9; ++q) rcell.cu[q] = c->cell_user[q];
    if (what == 0) {
        k_stage_copy0<<<nb, T, 0, c->stream>>>(c->n, c->orig, c->n_user, c->pos, c->vel, c->rep_stage);
        k_spread_copy0<<<nb, T, 0, c->stream>>>(c->n, c->orig, c->n_user, c->rep_m[0], c->rep_m[1], rcell, c->rep_stage, c->pos, c->vel, 1);
    } else {
        k_stage_copy0<<<nb, T, 0, c->stream>>>(c->n, c->orig, c->n_user, c->frc, nullptr, c->rep_stage);
        k_spread_copy0<<<nb, T, 0, c->stream>>>(c->n, c->orig, c->n_user, c->rep_m[0], c->rep_m[1], rcell, c->rep_stage, c->frc, nullptr, 0);
    }
    c->launches += 2;
    return NNP_OK;
}

void nnp_launch_unpermute3x2(nnp_ctx *c, const float4 *srcA, float *dstA, const float4 *srcB, float *dstB)
{
    k_unpermute3x2<<<nnp_div_up(c->n, T), T, 0, c->stream>>>(c->n, srcA, srcB, c->orig, c->n_user, dstA, dstB);
    c->launches += 1;
}

void nnp_launch_permute_in3x2(nnp_ctx *c, const float *srcA, float4 *dstA, const float *srcB, float4 *dstB)
{
    k_permute_in3x2<<<nnp_div_up(c->n, T), T, 0, c->stream>>>(c->n, srcA, srcB, c->orig, c->n_user, dstA, dstB);
    c->launches += 1;
}

void nnp_launch_pack_result(nnp_ctx *c)
{
    k_pack_result<<<1, 32, 0, c->stream>>>(c->e_mol, c->ekin, c->flags, c->d_res);
    c->launches += 1;
}

void nnp_launch_kick_drift(nnp_ctx *c)
{
    const float hs = 0.5f * c->skin;
    if (c->lgv_gamma > 0.f) {
        k_kick_drift_langevin<<<nnp_div_up(c->n, T), T, 0, c->stream>>>(
            c->n, c->pos, c->vel, c->frc, c->xref, c->spc, c->orig, c->d_inv_mass_conv, c->d_lgv_c2, c->lgv_c1, c->dt, hs * hs,
            (uint32_t)c->lgv_seed, (uint32_t)(c->lgv_seed >> 32), c->flags, c->n_user);
        c->launches += 1;
        nnp_launch_sync_copies(c, 0);
        return;
    }
    k_kick_drift<<<nnp_div_up(c->n, T), T, 0, c->stream>>>(c->n, c->pos, c->vel, c->frc, c->xref, c->spc,
                                                          c->d_inv_mass_conv, c->dt, hs * hs, c->flags);
    c->launches += 1;
    nnp_launch_sync_copies(c, 0);
}

void nnp_launch_kick_ke(nnp_ctx *c, int count_step)
{
    nnp_launch_sync_copies(c, 1); // (replicated small cell: every copy is kicked with its atom's force)
    cudaMemsetAsync(c->ekin, 0, sizeof(double) * c->n_mols, c->stream);
    k_kick_ke<<<nnp_div_up(c->n, T), T, 0, c->stream>>>(c->n, c->vel, c->frc, c->spc, c->d_inv_mass_conv, c->d_mass,
                                                       c->dt, 1.0f / c->accel_conv, 1.0f / (float)c->rep, c->mol, c->n_mols == 1, c->ekin,
                                                       count_step ? c->flags + 4 : nullptr);
    c->launches += 1;
}

void nnp_launch_energy_reduce(nnp_ctx *c)
{
    cudaMemsetAsync(c->e_mol, 0, sizeof(double) * c->n_mols, c->stream);
    k_energy_reduce<<<nnp_div_up(c->n, T), T, 0, c->stream>>>(c->n, c->e_atom, c->spc, c->mol, c->d_e_shift,
                                                             1.0f / (float)c->n_nets, 1.0 / (double)c->rep, c->n_mols == 1, c->e_mol);
    c->launches += 1;
}

void nnp_launch_unpermute3(nnp_ctx *c, const float4 *src, float *dst)
{
    k_unpermute3<<<nnp_div_up(c->n, T), T, 0, c->stream>>>(c->n, src, c->orig, c->n_user, dst);
    c->launches += 1;
}

void nnp_launch_permute_in3(nnp_ctx *c, const float *src, float4 *dst)
{
    k_permute_in3<<<nnp_div_up(c->n, T), T, 0, c->stream>>>(c->n, src, c->orig, c->n_user, dst);
    c->launches += 1;
}
