// C-ABI entry points (include/nnp.h): argument checking, device memory, and the order in which the stage
// kernels are enqueued.  Every arithmetic step of the path runs in the kernels of neighbor.cu, aev.cu,
// mlp_simt.cu / mlp_tc.cu and integrate.cu.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <vector>

#include "nnp_internal.cuh"

static std::string g_create_error;

#define NNP_FAIL(ctx, code, ...)                              \
    do {                                                      \
        char _b[512];                                         \
        snprintf(_b, sizeof(_b), __VA_ARGS__);                \
        if (ctx) (ctx)->err = _b; else g_create_error = _b;   \
        return (code);                                        \
    } while (0)

#define CU(ctx, call)                                                                              \
    do {                                                                                           \
        cudaError_t _e = (call);                                                                   \
        if (_e != cudaSuccess)                                                                     \
            NNP_FAIL(ctx, _e == cudaErrorMemoryAllocation ? NNP_ENOMEM : NNP_ECUDA, "%s: %s", #call, \
                     cudaGetErrorString(_e));                                                      \
    } while (0)

void nnp_prof_mark(nnp_ctx *c, int stage)
{
    if (!c->prof_active) return;
    cudaEvent_t ev;
    if (!c->prof_pool.empty()) { ev = c->prof_pool.back(); c->prof_pool.pop_back(); }
    else if (cudaEventCreate(&ev) != cudaSuccess) return;
    cudaEventRecord(ev, c->stream);
    c->prof_marks.emplace_back(ev, stage);
}

static void prof_begin(nnp_ctx *c)
{
    c->prof_active = c->prof_stride > 0 && (c->prof_calls++ % c->prof_stride) == 0 && c->prof_marks.size() < 200000;
    nnp_prof_mark(c, -1);
}

static void prof_collect(nnp_ctx *c)
{
    cudaStreamSynchronize(c->stream);
    for (size_t q = 0; q < c->prof_marks.size(); ++q) {
        const int st = c->prof_marks[q].second;
        if (st >= 0 && q > 0) {
            float ms = 0.f;
            if (cudaEventElapsedTime(&ms, c->prof_marks[q - 1].first, c->prof_marks[q].first) == cudaSuccess) {
                c->prof_ms[st] += ms;
            }
        }
    }
    // samples: one per "begin" mark for every stage that appeared after it
    int seen[NNP_N_STAGES];
    for (size_t q = 0; q < c->prof_marks.size(); ++q) {
        const int st = c->prof_marks[q].second;
        if (st < 0) { for (int k = 0; k < NNP_N_STAGES; ++k) seen[k] = 0; }
        else if (!seen[st]) { seen[st] = 1; c->prof_n[st] += 1; }
        c->prof_pool.push_back(c->prof_marks[q].first);
    }
    c->prof_marks.clear();
}

namespace {

constexpr int T = 256;

void cross3f(const double *u, const double *v, double *o)
{
    o[0] = u[1] * v[2] - u[2] * v[1]; o[1] = u[2] * v[0] - u[0] * v[2]; o[2] = u[0] * v[1] - u[1] * v[0];
}

// Copy m = (m0, m1, m2) of a replicated small cell: shift m0 a + m1 b + m2 c of the caller's cell (rows of cu).
struct RepInfo { int n_user, m[3]; float cu[9]; };
__device__ __forceinline__ float3 rep_shift(const RepInfo &r, int copy)
{
    const int m0 = copy % r.m[0], m1 = (copy / r.m[0]) % r.m[1], m2 = copy / (r.m[0] * r.m[1]);
    return make_float3((float)m0 * r.cu[0] + (float)m1 * r.cu[3] + (float)m2 * r.cu[6],
                       (float)m0 * r.cu[1] + (float)m1 * r.cu[4] + (float)m2 * r.cu[7],
                       (float)m0 * r.cu[2] + (float)m1 * r.cu[5] + (float)m2 * r.cu[8]);
}

__global__ void k_init_system(int n, const int *__restrict__ species, const float *__restrict__ xyz,
                              const int *__restrict__ mol_offsets, int n_mols, float4 *__restrict__ pos,
                              float4 *__restrict__ vel, int *__restrict__ spc, int *__restrict__ orig,
                              int *__restrict__ mol, int *__restrict__ counts, int S, int *__restrict__ bad, RepInfo rep)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (rep.n_user < n) { // replicated cell (one structure): internal atom e = copy * n_user + a
        if (i >= n) return;
        const int a = i % rep.n_user;
        const float3 sh = rep_shift(rep, i / rep.n_user);
        int s = species[a];
        if (s < 0 || s >= S) { atomicOr(bad, 1); s = 0; }
        pos[i] = make_float4(xyz[3 * a] + sh.x, xyz[3 * a + 1] + sh.y, xyz[3 * a + 2] + sh.z, 0.f);
        vel[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        spc[i] = s;
        orig[i] = i;
        mol[i] = 0;
        atomicAdd(&counts[s], 1);
        return;
    }
    if (mol_offsets) { // offsets[0] = 0 <= offsets[1] <= ... <= offsets[n_mols] = n, checked by a grid-stride loop
        for (int m = i; m <= n_mols; m += gridDim.x * blockDim.x) {
            const int o = mol_offsets[m];
            const bool ok = m == 0 ? o == 0 : (o >= mol_offsets[m - 1] && (m < n_mols || o == n));
            if (!ok) atomicOr(bad, 2);
        }
    }
    if (i >= n) return;
    int s = species[i];
    if (s < 0 || s >= S) { atomicOr(bad, 1); s = 0; }
    pos[i] = make_float4(xyz[3 * i], xyz[3 * i + 1], xyz[3 * i + 2], 0.f);
    vel[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    spc[i] = s;
    orig[i] = i;
    int m = 0;
    if (mol_offsets) { // largest m with mol_offsets[m] <= i
        int lo = 0, hi = n_mols;
        while (hi - lo > 1) { int mid = (lo + hi) >> 1; if (mol_offsets[mid] <= i) lo = mid; else hi = mid; }
        m = lo;
    }
    mol[i] = m;
    atomicAdd(&counts[s], 1);
}

__global__ void k_set_positions_rep(int n, const float *__restrict__ src, const int *__restrict__ orig, float4 *__restrict__ dst,
                                    RepInfo rep)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int e = orig[i], a = e % rep.n_user;
    const float3 sh = rep_shift(rep, e / rep.n_user);
    dst[i] = make_float4(src[3 * a] + sh.x, src[3 * a + 1] + sh.y, src[3 * a + 2] + sh.z, 0.f);
}

// rows of the caller's atoms (copies 0 of a replicated cell); an image of atom j is reported as j
__global__ void k_get_neighbors(int n, const int *__restrict__ nbr, const uint16_t *__restrict__ seg, int cap,
                                const int *__restrict__ orig, int n_user, int *__restrict__ counts, int *__restrict__ list,
                                int stride)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int o = orig[i];
    if (o >= n_user) return;
    const int cnt = seg[(size_t)i * NNP_MAX_SPECIES + NNP_MAX_SPECIES - 1];
    counts[o] = cnt;
    for (int a = 0; a < cnt && a < stride; ++a) list[(size_t)o * stride + a] = orig[nbr[(size_t)i * cap + a]] % n_user;
}

// Test hook: active columns of G -> the full aev_len layout (columns of absent species are zero).
__global__ void k_get_aev(int n, int len_full, int len_c, int kpad, const float *__restrict__ G, const int *__restrict__ fmap,
                          const int *__restrict__ orig, int n_user, float *__restrict__ out)
{
    int i = blockIdx.x;
    if (i >= n) return;
    const int o = orig[i];
    if (o >= n_user) return;
    for (int q = threadIdx.x; q < len_full; q += blockDim.x) out[(size_t)o * len_full + q] = 0.f;
    __syncthreads();
    for (int q = threadIdx.x; q < len_c; q += blockDim.x) out[(size_t)o * len_full + fmap[q]] = G[(size_t)i * kpad + q];
}

// Layer-1 weights restricted to the active AEV columns: row c of the compact matrix is row fmap[c] of the full one
// (zero for padding), in both orientations and, for the tensor-core modes, as tf32 hi / lo splits.
__global__ void k_gather_l1(int kpad, int out, const int *__restrict__ fmap, const float *__restrict__ W_full,
                            float *__restrict__ W, float *__restrict__ Wt, float *__restrict__ W_hi, float *__restrict__ W_lo,
                            float *__restrict__ Wt_hi, float *__restrict__ Wt_lo)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= kpad * out) return;
    const int c = idx / out, j = idx - c * out;
    const int f = fmap[c];
    const float v = f >= 0 ? W_full[(size_t)f * out + j] : 0.f;
    W[idx] = v;
    Wt[(size_t)j * kpad + c] = v;
    if (W_hi) {
        const uint32_t h = (__float_as_uint(v) + 0x1000u) & 0xffffe000u;
        const uint32_t l = (__float_as_uint(v - __uint_as_float(h)) + 0x1000u) & 0xffffe000u;
        W_hi[idx] = __uint_as_float(h); W_lo[idx] = __uint_as_float(l);
        Wt_hi[(size_t)j * kpad + c] = __uint_as_float(h); Wt_lo[(size_t)j * kpad + c] = __uint_as_float(l);
    }
}

__global__ void k_get_e_atom(int n, const float *__restrict__ e_atom, const int *__restrict__ spc,
                             const float *__restrict__ e_shift, float inv_nets, const int *__restrict__ orig, int n_user,
                             float *__restrict__ out)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n || orig[i] >= n_user) return;
    out[orig[i]] = e_atom[i] * inv_nets + e_shift[spc[i]];
}

// Sets the IF node of the MD-step graph from the rebuild request the drift kernel left in flags[1].
__global__ void k_set_rebuild_cond(cudaGraphConditionalHandle h, const int *__restrict__ flag)
{
    cudaGraphSetConditional(h, *flag != 0 ? 1u : 0u);
}

// Every device buffer of the library comes from here: the caller's allocator (nnp_params.alloc, e.g. PyTorch's caching
// allocator) or cudaMalloc.
template <typename Tp>
int dev_alloc(nnp_ctx *c, Tp **p, size_t count)
{
    const size_t bytes = sizeof(Tp) * (count ? count : 1);
    if (c->alloc_fn) {
        *p = (Tp *)c->alloc_fn(bytes, c->alloc_user);
        if (!*p) NNP_FAIL(c, NNP_ENOMEM, "nnp_params.alloc(%zu bytes) returned NULL", bytes);
        if ((uintptr_t)*p & 255u) NNP_FAIL(c, NNP_EINVAL, "nnp_params.alloc returned a pointer that is not 256-byte aligned");
        return NNP_OK;
    }
    CU(c, cudaMalloc((void **)p, bytes));
    return NNP_OK;
}
void dev_free(nnp_ctx *c, void *p)
{
    if (!p) return;
    if (c->dealloc_fn) c->dealloc_fn(p, c->alloc_user);
    else cudaFree(p);
}

LayerW &layer(nnp_ctx *c, int net, int s, int l) { return c->layers[((size_t)net * c->S + s) * NNP_NLAYERS + l]; }
Layer1C &l1c(nnp_ctx *c, int net, int s) { return c->l1c[(size_t)net * c->S + s]; }

// Active-column layout for the species in `mask`; rebuilds the compact layer-1 copies when the mask changed.
int set_layout(nnp_ctx *c, unsigned mask)
{
    AevParams &a = c->aev;
    const int S = c->S;
    int np = 0;
    for (int s = 0; s < NNP_MAX_SPECIES; ++s) { a.cmap[s] = -1; a.plist[s] = 0; }
    for (int s = 0; s < S; ++s)
        if (mask >> s & 1u) { a.cmap[s] = np; a.plist[np] = s; ++np; }
    a.np = np;
    a.n_rad = np * NNP_NSHF_R;
    a.aev_len = a.n_rad + np * (np + 1) / 2 * NNP_ANG_BLOCK;
    a.kpad = (a.aev_len + 31) / 32 * 32;
    if (mask == c->present_mask) return NNP_OK;
    // compact column -> full column
    std::vector<int> fmap(c->kpad_full, -1);
    for (int cs = 0; cs < np; ++cs)
        for (int k = 0; k < NNP_NSHF_R; ++k) fmap[cs * NNP_NSHF_R + k] = a.plist[cs] * NNP_NSHF_R + k;
    int pc = 0;
    for (int cs = 0; cs < np; ++cs)
        for (int ct = cs; ct < np; ++ct, ++pc) {
            const int s = a.plist[cs], t = a.plist[ct];
            const int pf = s * (2 * S + 1 - s) / 2 + (t - s);
            for (int q = 0; q < NNP_ANG_BLOCK; ++q) fmap[a.n_rad + pc * NNP_ANG_BLOCK + q] = S * NNP_NSHF_R + pf * NNP_ANG_BLOCK + q;
        }
    CU(c, cudaMemcpyAsync(c->d_fmap, fmap.data(), sizeof(int) * c->kpad_full, cudaMemcpyHostToDevice, c->stream));
    CU(c, cudaStreamSynchronize(c->stream)); // fmap is a stack-lifetime host buffer
    float *base = c->d_l1c_blob;
    const int narr = c->tc_mode ? 6 : 2;
    for (int net = 0; net < c->n_nets; ++net)
        for (int s = 0; s < S; ++s) {
            const int out = c->widths[s][1];
            const size_t cnt = (size_t)a.kpad * out;
            Layer1C &L = l1c(c, net, s);
            L.W = base; L.Wt = base + cnt;
            L.W_hi = L.W_lo = L.Wt_hi = L.Wt_lo = nullptr;
            if (c->tc_mode) { L.W_hi = base + 2 * cnt; L.W_lo = base + 3 * cnt; L.Wt_hi = base + 4 * cnt; L.Wt_lo = base + 5 * cnt; }
            base += (size_t)narr * c->kpad_full * out;
            k_gather_l1<<<nnp_div_up((int)cnt, T), T, 0, c->stream>>>(a.kpad, out, c->d_fmap, layer(c, net, s, 0).W, L.W, L.Wt,
                                                                      L.W_hi, L.W_lo, L.Wt_hi, L.Wt_lo);
            c->launches += 1;
        }
    // G / dG: columns beyond aev_len must be zero (layer 1 multiplies all kpad columns)
    CU(c, cudaMemsetAsync(c->G, 0, sizeof(float) * (size_t)c->max_atoms * c->kpad_full, c->stream));
    CU(c, cudaGetLastError());
    c->present_mask = mask;
    return NNP_OK;
}

// Gaussian ladder constants (AevParams::ladder).  Shift k = 4m + J of group m relative to the anchor a = 4m + 1:
//   2^-(w_a - (k-a) d)^2 = 2^-(w_a^2) * 2^(2 (k-a) d w_0) * 2^(-(k-a) d^2 (2 (a-1) + (k-a))),  w_a = w_0 - (a-1) d,
// the last factor is lad[k].  Used only if the shifts are uniform to fp32 accuracy and every intermediate power
// stays well inside the fp32 exponent range for r up to the cutoff; NNP_NO_LADDER=1 forces the direct evaluation.
void setup_ladder(AevParams &a, const nnp_params *p)
{
    auto uniform = [](const float *shf, int n, double &step) {
        step = ((double)shf[n - 1] - (double)shf[0]) / (n - 1);
        if (!(step > 0.0)) return false;
        for (int k = 0; k < n; ++k)
            if (fabs((double)shf[k] - ((double)shf[0] + k * step)) > 2.5e-7 * fabs((double)shf[n - 1])) return false;
        return true;
    };
    double step_r = 0.0, step_a = 0.0;
    bool ok = uniform(p->shf_r, NNP_NSHF_R, step_r) && uniform(p->shf_a, NNP_NSHF_A, step_a);
    const double kr = sqrt((double)p->eta_r * 1.4426950408889634), ka = sqrt((double)p->eta_a * 1.4426950408889634);
    const double dr = kr * step_r, da = ka * step_a;
    if (ok) {
        // largest exponents met: Q^2 = 2^(4 d w_0max), raw sums 2^((4 + 16 m_max) d^2); smallest: 2^(-2 d w_0max - ...)
        const double w0r = kr * ((double)p->rcr - (double)p->shf_r[1]), w0a = ka * ((double)p->rca - (double)p->shf_a[1]);
        const double lim = 125.0; // fp32 overflows at 2^128
        ok = 4.0 * dr * w0r < lim && 4.0 * da * w0a < lim && (4.0 + 16.0 * (NNP_NSHF_R / 4 - 1)) * dr * dr < lim - 8.0 &&
             (4.0 + 16.0 * (NNP_NSHF_A / 4 - 1)) * da * da < lim - 8.0 && p->shf_r[1] > 0.f && p->shf_a[1] > 0.f;
    }
    const char *env = getenv("NNP_NO_LADDER");
    if (env && env[0] == '1') ok = false;
    a.ladder = ok ? 1 : 0;
    a.dlt_r = (float)dr; a.dlt_a = (float)da;
    for (int k = 0; k < NNP_NSHF_R; ++k) {
        const int an = 4 * (k / 4) + 1, j = k - an;
        a.lad_r[k] = ok ? (float)exp2(-(double)j * dr * dr * (2.0 * (an - 1) + j)) : 1.0f;
    }
    for (int k = 0; k < NNP_NSHF_A; ++k) {
        const int an = 4 * (k / 4) + 1, j = k - an;
        a.lad_a[k] = ok ? (float)exp2(-(double)j * da * da * (2.0 * (an - 1) + j)) : 1.0f;
    }
}

} // namespace

void nnp_aev_derive(AevParams &a)
{
    for (int z = 0; z < NNP_NSHF_Z / 2; ++z) {
        a.hcz2[z] = make_float2(0.5f * a.cos_z[2 * z], 0.5f * a.cos_z[2 * z + 1]);
        a.hsz2[z] = make_float2(0.5f * a.sin_z[2 * z], 0.5f * a.sin_z[2 * z + 1]);
        a.nhsz2[z] = make_float2(-0.5f * a.sin_z[2 * z], -0.5f * a.sin_z[2 * z + 1]);
    }
    for (int k = 0; k < NNP_NSHF_A / 2; ++k) a.nka_shf2[k] = make_float2(-a.ka_shf[2 * k], -a.ka_shf[2 * k + 1]);
    for (int k = 0; k < NNP_NSHF_R / 2; ++k) a.nkr_shf2[k] = make_float2(-a.kr_shf[2 * k], -a.kr_shf[2 * k + 1]);
    for (int m = 0; m < NNP_NSHF_R / 8; ++m) a.nkr_anc2[m] = make_float2(-a.kr_shf[8 * m + 1], -a.kr_shf[8 * m + 5]);
    a.nka_anc2 = make_float2(-a.ka_shf[1], -a.ka_shf[5]);
    a.half_ka = 0.5f * a.ka;
    a.k_ang0 = 0.5f * a.zeta * 0.95f * 2.0f;
    a.zm1 = a.zeta - 1.0f;
    a.half_drb_scale = 0.5f * (-2.0f * a.eta_a / a.ka);
    a.dr_scale = -2.0f * a.eta_r / a.kr;
    a.nh_pi_rcr = -0.5f * a.pi_rcr;
    a.nh_pi_rca = -0.5f * a.pi_rca;
    a.two_dlt_r = 2.0f * a.dlt_r;
    a.two_dlt_a = 2.0f * a.dlt_a;
}

namespace {

int check_flags(nnp_ctx *c)
{
    int h[3];
    CU(c, cudaMemcpyAsync(h, c->flags, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    if (h[0] & (NNP_FLAG_CAP_R | NNP_FLAG_CAP_A))
        NNP_FAIL(c, NNP_ECAPACITY, "neighbour capacity exceeded (%s): recreate with larger cap_r/cap_a",
                 (h[0] & NNP_FLAG_CAP_R) ? "radial" : "angular");
    if (h[0] & NNP_FLAG_RANGE)
        NNP_FAIL(c, NNP_ERANGE, "mm_mode 4: an activation exceeded the range of the scaled fp16 split; use mm_mode 1");
    return NNP_OK;
}

// One GemmBatch per op and range of networks [net0, net0 + n_batch): one group per (network, species present); op 0..2
// forward layers, 3..5 reverse layers.  Every network of an ensemble has its own activation buffers, so the layers of
// several networks run as ONE grouped launch (a 12k-atom ensemble call is otherwise 48 launches of ~100 tiles).
void make_batch(nnp_ctx *c, int net0, int n_batch, int op, GemmBatch &b)
{
    memset(&b, 0, sizeof(b));
    b.alpha = c->alpha;
    const int kpad = c->aev.kpad;
    int ng = 0;
    for (int net = net0; net < net0 + n_batch; ++net)
    for (int s = 0; s < c->S; ++s) {
        const int off = c->bucket_off[s], M = c->bucket_off[s + 1] - off;
        if (M == 0) continue;
        GemmGroup &g = b.g[ng++];
        const int h1 = c->widths[s][1], h2 = c->widths[s][2], h3 = c->widths[s][3];
        float *H0 = c->H[0] + ((size_t)net * c->max_atoms + off) * c->hmax[0];
        float *H1 = c->H[1] + ((size_t)net * c->max_atoms + off) * c->hmax[1];
        float *H2 = c->H[2] + ((size_t)net * c->max_atoms + off) * c->hmax[2];
        g.M = M;
        switch (op) {
        case 0:
            g.A = c->G + (size_t)off * kpad; g.lda = kpad; g.K = kpad; g.N = h1;
            g.B = l1c(c, net, s).W; g.Bt = l1c(c, net, s).Wt; g.bias = layer(c, net, s, 0).b;
            g.Bt_hi = l1c(c, net, s).Wt_hi; g.Bt_lo = l1c(c, net, s).Wt_lo;
            g.C = H0; g.ldc = c->hmax[0];
            break;
        case 1:
            g.A = H0; g.lda = c->hmax[0]; g.K = h1; g.N = h2;
            g.B = layer(c, net, s, 1).W; g.Bt = layer(c, net, s, 1).Wt; g.bias = layer(c, net, s, 1).b;
            g.Bt_hi = layer(c, net, s, 1).Wt_hi; g.Bt_lo = layer(c, net, s, 1).Wt_lo;
            g.C = H1; g.ldc = c->hmax[1];
            break;
        case 2:
            g.A = H1; g.lda = c->hmax[1]; g.K = h2; g.N = h3;
            g.B = layer(c, net, s, 2).W; g.Bt = layer(c, net, s, 2).Wt; g.bias = layer(c, net, s, 2).b;
            g.Bt_hi = layer(c, net, s, 2).Wt_hi; g.Bt_lo = layer(c, net, s, 2).Wt_lo;
            g.w4 = layer(c, net, s, 3).W; g.e_atom = c->e_atom + off;
            g.C = H2; g.ldc = c->hmax[2];
            break;
        case 3: // delta2 = (delta3 W3^T) * celu'(h2), in place in H1
            g.A = H2; g.lda = c->hmax[2]; g.K = h3; g.N = h2;
            g.B = layer(c, net, s, 2).Wt; g.Bt = layer(c, net, s, 2).W;
            g.Bt_hi = layer(c, net, s, 2).W_hi; g.Bt_lo = layer(c, net, s, 2).W_lo;
            g.C = H1; g.ldc = c->hmax[1];
            break;
        case 4: // delta1 = (delta2 W2^T) * celu'(h1), in place in H0
            g.A = H1; g.lda = c->hmax[1]; g.K = h2; g.N = h1;
            g.B = layer(c, net, s, 1).Wt; g.Bt = layer(c, net, s, 1).W;
            g.Bt_hi = layer(c, net, s, 1).W_hi; g.Bt_lo = layer(c, net, s, 1).W_lo;
            g.C = H0; g.ldc = c->hmax[0];
            break;
        case 5: // dE/dG (+)= delta1 W1^T
            g.A = H0; g.lda = c->hmax[0]; g.K = h1; g.N = kpad;
            g.B = l1c(c, net, s).Wt; g.Bt = l1c(c, net, s).W;
            g.Bt_hi = l1c(c, net, s).W_hi; g.Bt_lo = l1c(c, net, s).W_lo;
            g.C = c->dG + (size_t)off * kpad; g.ldc = kpad;
            break;
        }
    }
    b.n_groups = ng;
}

int run_gemm(nnp_ctx *c, const GemmBatch &b, int epi)
{
    if (!c->tc_mode) { nnp_launch_gemm_simt(c, b, epi, c->mm_mode == NNP_MM_FP64_SIMT); return NNP_OK; }
    return nnp_launch_gemm_tc(c, b, epi, c->split3);
}

// Stages 2-4 on the current lists: frc, e_mol.
int run_forces(nnp_ctx *c)
{
    CU(c, cudaMemsetAsync(c->frc, 0, sizeof(float4) * (size_t)c->n, c->stream));
    CU(c, cudaMemsetAsync(c->e_atom, 0, sizeof(float) * (size_t)c->n, c->stream));
    nnp_launch_aev_forward(c);
    nnp_prof_mark(c, 2);
    static const int epi_of[6] = {EPI_CELU, EPI_CELU, EPI_CELU_OUT, EPI_DCELU, EPI_DCELU, EPI_STORE};
    GemmBatch b;
    // networks per grouped launch (tensor-core modes): as many as the group table holds
    const int np = c->aev.np > 0 ? c->aev.np : 1;
    int nb = (!c->tc_mode || c->n_nets == 1) ? 1 : NNP_MAX_GROUPS / np;
    if (nb < 1) nb = 1;
    if (nb > c->n_nets) nb = c->n_nets;
    // mm_mode 4: all six GEMMs of every network and species in one launch (mlp_fused.cu); nnp_fused_kind is 0 where the chain
    // does not apply (hidden widths outside [64, 256], more than 64 (network, species) groups): six 3xTF32 launches then
    if (nnp_fused_kind(c) == 1) {
        if (c->n_nets > 1) CU(c, cudaMemsetAsync(c->dG, 0, sizeof(float) * (size_t)c->n * c->aev.kpad, c->stream));
        nnp_launch_mlp_fused(c);
        nnp_prof_mark(c, 12);
    } else {
        for (int net0 = 0; net0 < c->n_nets; net0 += nb)
            for (int op = 0; op < 5; ++op) {
                make_batch(c, net0, nb < c->n_nets - net0 ? nb : c->n_nets - net0, op, b);
                int rc = run_gemm(c, b, epi_of[op]);
                if (rc != NNP_OK) return rc;
                nnp_prof_mark(c, 3 + op);
            }
        if (nb > 1) {
            // dE/dG sums over the networks: the groups of all batched networks add into the same rows with vector
            // reductions in memory (the summation order over the networks is then not fixed, like the force scatter's)
            CU(c, cudaMemsetAsync(c->dG, 0, sizeof(float) * (size_t)c->n * c->aev.kpad, c->stream));
            for (int net0 = 0; net0 < c->n_nets; net0 += nb) {
                make_batch(c, net0, nb < c->n_nets - net0 ? nb : c->n_nets - net0, 5, b);
                int rc = run_gemm(c, b, EPI_RED);
                if (rc != NNP_OK) return rc;
                nnp_prof_mark(c, 8);
            }
        } else {
            for (int net = 0; net < c->n_nets; ++net) { // one network per launch, accumulated in place in network order
                make_batch(c, net, 1, 5, b);
                int rc = run_gemm(c, b, net > 0 ? EPI_ACCUM : EPI_STORE);
                if (rc != NNP_OK) return rc;
                nnp_prof_mark(c, 8);
            }
        }
    }
    nnp_launch_energy_reduce(c);
    nnp_prof_mark(c, 9);
    nnp_launch_aev_backward(c, 1.0f / (float)c->n_nets, c->want_virial ? c->d_virial : nullptr);
    nnp_prof_mark(c, 10);
    CU(c, cudaGetLastError());
    c->have_forces = 1;
    return NNP_OK;
}

int setup_grid(nnp_ctx *c, float skin)
{
    GridInfo &g = c->grid;
    memset(&g, 0, sizeof(g));
    const float rl = c->aev.rcr + skin;
    g.periodic = c->periodic;
    if (c->periodic) {
        long ncell = 1;
        double h[9], rec[9];
        for (int q = 0; q < 9; ++q) h[q] = c->cell[q];
        cross3f(h + 3, h + 6, rec); cross3f(h + 6, h, rec + 3); cross3f(h, h + 3, rec + 6);
        const double vol = h[0] * rec[0] + h[1] * rec[1] + h[2] * rec[2];
        g.tric = c->tric;
        for (int q = 0; q < 9; ++q) { g.h[q] = c->cell[q]; g.hinv[q] = (float)(rec[q] / vol); }
        for (int d = 0; d < 3; ++d) {
            // perpendicular width of the (super)cell along lattice direction d (= the edge of an orthorhombic box)
            const float w = c->tric ? (float)(fabs(vol) / sqrt(rec[3 * d] * rec[3 * d] + rec[3 * d + 1] * rec[3 * d + 1] + rec[3 * d + 2] * rec[3 * d + 2]))
                                    : c->box[d];
            if (w < 2.0f * rl)
                NNP_FAIL(c, NNP_EBOX, "cell width %g < 2*(rcr+skin) = %g: minimum image not unique%s", w, 2.0f * rl,
                         c->rep > 1 ? " (the supercell of a small cell is sized for a skin of 0.5 A)" : "");
            int nc = (int)floorf(w / (rl * 1.0001f));
            if (nc < 1) nc = 1;
            if (nc > 128) nc = 128;
            g.nc[d] = nc;
            g.box[d] = c->box[d];
            g.inv_box[d] = 1.0f / c->box[d];
            g.cell_scale[d] = c->tric ? (float)nc : (float)nc / c->box[d];
            ncell *= nc;
        }
        // a periodic batch (replicas of one cell, e.g. the beads of a ring polymer): one bin set per replica
        if (ncell * c->n_mols * c->S > (1L << 27))
            NNP_FAIL(c, NNP_EINVAL, "%ld cells x %d structures x %d species: too many bins", ncell, c->n_mols, c->S);
        g.ncell_box = (int)ncell;
        g.ncell = (int)ncell * c->n_mols;
    } else {
        g.nc[0] = c->n_mols; g.nc[1] = 1; g.nc[2] = 1;
        g.ncell = c->n_mols;
    }
    const int nk = c->S * g.ncell + 1;
    if (nk > c->nkeys_cap) {
        CU(c, cudaStreamSynchronize(c->stream)); // earlier builds may still read the old arrays
        dev_free(c, c->cell_start);
        dev_free(c, c->cursor);
        c->cell_start = c->cursor = nullptr;
        c->nkeys_cap = 0;
        int rc;
        if ((rc = dev_alloc(c, &c->cell_start, nk))) return rc;
        if ((rc = dev_alloc(c, &c->cursor, nk))) return rc;
        c->nkeys_cap = nk;
    }
    CU(c, cudaMemsetAsync(c->cursor, 0, sizeof(int) * nk, c->stream));
    c->aev.periodic = c->periodic;
    c->aev.tric = g.tric;
    for (int d = 0; d < 3; ++d) { c->aev.box[d] = g.box[d]; c->aev.inv_box[d] = g.inv_box[d]; }
    for (int q = 0; q < 9; ++q) { c->aev.h[q] = g.h[q]; c->aev.hinv[q] = g.hinv[q]; }
    return NNP_OK;
}

void drop_md_graph(nnp_ctx *c)
{
    if (c->md_exec) { cudaGraphExecDestroy(c->md_exec); c->md_exec = nullptr; }
    if (c->md_graph) { cudaGraphDestroy(c->md_graph); c->md_graph = nullptr; }
}

// Captures one MD step into a graph.  The neighbour rebuild (8 kernels) sits in the body of a conditional IF node
// whose value a one-thread kernel copies from the device-side rebuild request, so a step without a rebuild
// launches none of them (the kernel-by-kernel path launches all 8 and lets each return at once).
int build_md_graph(nnp_ctx *c)
{
    drop_md_graph(c);
    if (!c->aux_stream) CU(c, cudaStreamCreateWithFlags(&c->aux_stream, cudaStreamNonBlocking));
    cudaGraph_t g = nullptr;
    CU(c, cudaGraphCreate(&g, 0));
    c->md_graph = g;
    cudaGraphConditionalHandle h;
    CU(c, cudaGraphConditionalHandleCreate(&h, g, 0, cudaGraphCondAssignDefault));
    const int64_t launches0 = c->launches;
    int rc = NNP_OK;
    cudaStream_t main_stream = c->stream;
    CU(c, cudaStreamBeginCaptureToGraph(main_stream, g, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal));
    bool capturing = true;
    do {
        nnp_launch_kick_drift(c);
        k_set_rebuild_cond<<<1, 1, 0, main_stream>>>(h, c->flags + 1);
        c->launches += 1;
        cudaStreamCaptureStatus st;
        const cudaGraphNode_t *deps = nullptr;
        size_t ndeps = 0;
        if (cudaStreamGetCaptureInfo_v2(main_stream, &st, nullptr, nullptr, &deps, &ndeps) != cudaSuccess) { rc = NNP_ECUDA; break; }
        cudaGraphNodeParams np = {cudaGraphNodeTypeConditional};
        np.conditional.handle = h;
        np.conditional.type = cudaGraphCondTypeIf;
        np.conditional.size = 1;
        cudaGraphNode_t cnode;
        if (cudaGraphAddNode(&cnode, g, deps, ndeps, &np) != cudaSuccess) { rc = NNP_ECUDA; break; }
        cudaGraph_t body = np.conditional.phGraph_out[0];
        const int64_t l1 = c->launches;
        if (cudaStreamBeginCaptureToGraph(c->aux_stream, body, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { rc = NNP_ECUDA; break; }
        c->stream = c->aux_stream;
        nnp_launch_build(c, nullptr);
        c->stream = main_stream;
        cudaGraph_t body_out = nullptr;
        if (cudaStreamEndCapture(c->aux_stream, &body_out) != cudaSuccess) { rc = NNP_ECUDA; break; }
        c->launches = l1; // the body's kernels run only on a rebuild: counted from the device-side rebuild counter
        if (cudaStreamUpdateCaptureDependencies(main_stream, &cnode, 1, cudaStreamSetCaptureDependencies) != cudaSuccess) { rc = NNP_ECUDA; break; }
        rc = run_forces(c);
        if (rc) break;
        nnp_launch_kick_ke(c, 1);
    } while (0);
    cudaGraph_t out = nullptr;
    cudaError_t e = capturing ? cudaStreamEndCapture(main_stream, &out) : cudaSuccess;
    c->stream = main_stream;
    c->md_graph_launches = c->launches - launches0;
    c->launches = launches0;
    if (rc == NNP_OK && e != cudaSuccess) rc = NNP_ECUDA;
    if (rc == NNP_OK && cudaGraphInstantiate(&c->md_exec, g, 0) != cudaSuccess) rc = NNP_ECUDA;
    if (rc != NNP_OK) {
        const cudaError_t last = cudaGetLastError();
        drop_md_graph(c);
        if (c->err.empty() || rc == NNP_ECUDA) c->err = std::string("MD-step graph capture failed: ") + cudaGetErrorString(last != cudaSuccess ? last : e);
    }
    return rc;
}

} // namespace

extern "C" {

const char *nnp_last_error(const nnp_ctx *ctx) { return ctx ? ctx->err.c_str() : g_create_error.c_str(); }

int64_t nnp_launch_count(const nnp_ctx *ctx) { return ctx ? ctx->launches : 0; }
int nnp_aev_len(const nnp_ctx *ctx) { return ctx ? ctx->aev_len_full : 0; }
int nnp_aev_active_columns(const nnp_ctx *ctx) { return ctx ? ctx->aev.aev_len : 0; }
int nnp_aev_ladder(const nnp_ctx *ctx) { return ctx ? ctx->aev.ladder : 0; }

void nnp_destroy(nnp_ctx *c)
{
    if (!c) return;
    cudaSetDevice(c->device);
    cudaStreamSynchronize(c->stream);
    drop_md_graph(c);
    nnp_fused_destroy(c);
    if (c->aux_stream) cudaStreamDestroy(c->aux_stream);
    void *ptrs[] = {c->d_params_blob, c->d_l1c_blob, c->d_fmap, c->d_tri, c->d_inv_mass_conv, c->d_mass, c->d_e_shift, c->d_lgv_c2, c->d_virial, c->pos, c->pos_tmp, c->vel, c->vel_tmp,
                    c->frc, c->xref, c->spc, c->spc_tmp, c->orig, c->orig_tmp, c->mol, c->mol_tmp, c->mol_offsets, c->key,
                    c->order, c->cell_start, c->cursor, c->nbr_r, c->nbr_a, c->seg_r, c->seg_a, c->G,
                    c->dG == c->G ? nullptr : c->dG, c->H[0], c->H[1], c->H[2], c->e_atom, c->e_mol, c->ekin, c->flags, c->aev_sched,
                    c->io_xyz, c->io_vel, c->io_species, c->d_res, c->rep_stage};
    for (void *p : ptrs) dev_free(c, p);
    if (c->h_res) cudaFreeHost(c->h_res);
    for (auto &m : c->prof_marks) cudaEventDestroy(m.first);
    for (auto &e : c->prof_pool) cudaEventDestroy(e);
    delete[] c->layers;
    delete[] c->l1c;
    delete c;
}

int nnp_create(nnp_ctx **out, const nnp_params *p, int max_atoms, int max_mols, int device, void *cuda_stream)
{
    nnp_ctx *none = nullptr;
    if (!out || !p) NNP_FAIL(none, NNP_EINVAL, "null argument");
    *out = nullptr;
    if (p->n_species < 1 || p->n_species > 7) NNP_FAIL(none, NNP_EINVAL, "n_species must be 1..7");
    if (p->n_shf_r != NNP_NSHF_R || p->n_shf_a != NNP_NSHF_A || p->n_shf_z != NNP_NSHF_Z || p->n_layers != NNP_NLAYERS)
        NNP_FAIL(none, NNP_EINVAL, "this build is fixed to 16 radial shifts, 8x4 angular shifts, 4 layers");
    if (!p->shf_r || !p->shf_a || !p->shf_z || !p->widths || !p->params || !p->mass)
        NNP_FAIL(none, NNP_EINVAL, "null parameter array");
    if (max_atoms < 1 || max_mols < 1 || p->n_nets < 1) NNP_FAIL(none, NNP_EINVAL, "max_atoms, max_mols, n_nets must be >= 1");
    if (!(p->rcr > 0.f) || !(p->rca > 0.f) || p->rca > p->rcr) NNP_FAIL(none, NNP_EINVAL, "need 0 < rca <= rcr");
    if (p->mm_mode < 0 || p->mm_mode > 4) NNP_FAIL(none, NNP_EINVAL, "bad mm_mode");
    if ((p->alloc == nullptr) != (p->dealloc == nullptr)) NNP_FAIL(none, NNP_EINVAL, "alloc and dealloc must be given together");
    const int S = p->n_species;
    const int aev_len = S * NNP_NSHF_R + S * (S + 1) / 2 * NNP_ANG_BLOCK;
    for (int s = 0; s < S; ++s) {
        const int *w = p->widths + s * (NNP_NLAYERS + 1);
        if (w[0] != aev_len || w[4] != 1) NNP_FAIL(none, NNP_EINVAL, "widths[%d] must start with %d and end with 1", s, aev_len);
        for (int l = 1; l <= 3; ++l)
            if (w[l] < 32 || w[l] > 256 || w[l] % 32) NNP_FAIL(none, NNP_EINVAL, "hidden widths must be multiples of 32 in [32,256]");
    }
    int cap_r = p->cap_r ? p->cap_r : 160, cap_a = p->cap_a ? p->cap_a : 64;
    if (cap_r < 4 || cap_r > 65532 || cap_r % 4 || cap_a < 4 || cap_a > 65532 || cap_a % 4)
        NNP_FAIL(none, NNP_EINVAL, "cap_r / cap_a must be multiples of 4");

    if (cudaSetDevice(device) != cudaSuccess) NNP_FAIL(none, NNP_ECUDA, "cudaSetDevice(%d) failed", device);
    nnp_ctx *c = new nnp_ctx();
    // new T() value-initialises: every POD member starts at zero
    c->S = S; c->n_nets = p->n_nets; c->mm_mode = p->mm_mode; c->tc_mode = p->mm_mode == NNP_MM_3XTF32_TC || p->mm_mode == NNP_MM_TF32_TC || p->mm_mode == NNP_MM_3XF16_TC; c->split3 = p->mm_mode != NNP_MM_TF32_TC; c->dense_aev = p->dense_aev != 0;
    c->alpha = p->celu_alpha; c->accel_conv = p->accel_conv;
    c->stream = (cudaStream_t)cuda_stream; c->device = device;
    c->alloc_fn = p->alloc; c->dealloc_fn = p->dealloc; c->alloc_user = p->alloc_user;
    { // the legacy / per-thread default streams cannot be captured: steps are then enqueued kernel by kernel
        const char *e = getenv("NNP_NO_GRAPH");
        c->no_graph = (e && e[0] == '1') || c->stream == nullptr || c->stream == cudaStreamLegacy || c->stream == cudaStreamPerThread;
        const char *f = getenv("NNP_NO_FUSED");
        c->no_fused = f && f[0] == '1';
    }
    c->max_atoms = max_atoms; c->max_mols = max_mols;
    c->hmax[0] = c->hmax[1] = c->hmax[2] = 0;
    for (int s = 0; s < S; ++s)
        for (int l = 0; l <= NNP_NLAYERS; ++l) {
            c->widths[s][l] = p->widths[s * (NNP_NLAYERS + 1) + l];
            if (l >= 1 && l <= 3 && c->widths[s][l] > c->hmax[l - 1]) c->hmax[l - 1] = c->widths[s][l];
        }
    AevParams &a = c->aev;
    a.S = S; a.n_rad = S * NNP_NSHF_R; a.aev_len = aev_len; a.kpad = (aev_len + 31) / 32 * 32;
    a.np = S;
    for (int s = 0; s < NNP_MAX_SPECIES; ++s) { a.cmap[s] = s < S ? s : -1; a.plist[s] = s < S ? s : 0; }
    c->aev_len_full = aev_len; c->kpad_full = a.kpad;
    a.cap_r = cap_r; a.cap_a = cap_a;
    a.rcr = p->rcr; a.rca = p->rca; a.rcr2 = p->rcr * p->rcr; a.rca2 = p->rca * p->rca;
    a.pi_rcr = (float)(M_PI / (double)p->rcr); a.pi_rca = (float)(M_PI / (double)p->rca);
    a.eta_r = p->eta_r; a.eta_a = p->eta_a; a.zeta = p->zeta;
    a.neg_eta_r_log2e = (float)(-(double)p->eta_r * 1.4426950408889634);
    a.neg_eta_a_log2e = (float)(-(double)p->eta_a * 1.4426950408889634);
    a.ka = (float)sqrt((double)p->eta_a * 1.4426950408889634);
    a.kr = (float)sqrt((double)p->eta_r * 1.4426950408889634);
    for (int k = 0; k < NNP_NSHF_R; ++k) a.kr_shf[k] = (float)(sqrt((double)p->eta_r * 1.4426950408889634) * (double)p->shf_r[k]);
    for (int k = 0; k < NNP_NSHF_A; ++k) a.ka_shf[k] = (float)(sqrt((double)p->eta_a * 1.4426950408889634) * (double)p->shf_a[k]);
    for (int k = 0; k < NNP_NSHF_R; ++k) a.shf_r[k] = p->shf_r[k];
    for (int k = 0; k < NNP_NSHF_A; ++k) a.shf_a[k] = p->shf_a[k];
    for (int k = 0; k < NNP_NSHF_Z; ++k) { a.cos_z[k] = (float)cos((double)p->shf_z[k]); a.sin_z[k] = (float)sin((double)p->shf_z[k]); }
    setup_ladder(a, p);
    nnp_aev_derive(a);

    // ---- weights: W [in_pad][out], Wt [out][in_pad], b [out] for every (net, species, layer)
    c->layers = new LayerW[(size_t)c->n_nets * S * NNP_NLAYERS];
    c->l1c = new Layer1C[(size_t)c->n_nets * S]();
    size_t total = 0, total_l1c = 0;
    for (int s = 0; s < S; ++s) total_l1c += (size_t)c->n_nets * (c->tc_mode ? 6 : 2) * a.kpad * c->widths[s][1];
    for (int net = 0; net < c->n_nets; ++net)
        for (int s = 0; s < S; ++s)
            for (int l = 0; l < NNP_NLAYERS; ++l) {
                LayerW &L = layer(c, net, s, l);
                L.in = c->widths[s][l]; L.out = c->widths[s][l + 1];
                L.in_pad = l == 0 ? a.kpad : L.in;
                total += (c->tc_mode ? 6 : 2) * (size_t)L.in_pad * L.out + (size_t)((L.out + 3) / 4 * 4);
            }
    std::vector<float> blob(total, 0.f);
    std::vector<double> shift(S, 0.0);
    {
        size_t o = 0;
        const float *src = p->params;
        for (int net = 0; net < c->n_nets; ++net)
            for (int s = 0; s < S; ++s)
                for (int l = 0; l < NNP_NLAYERS; ++l) {
                    LayerW &L = layer(c, net, s, l);
                    float *W = &blob[o]; o += (size_t)L.in_pad * L.out;
                    float *Wt = &blob[o]; o += (size_t)L.in_pad * L.out;
                    float *b = &blob[o]; o += (size_t)((L.out + 3) / 4 * 4);
                    L.wmax = 0.f;
                    for (int i = 0; i < L.in; ++i)
                        for (int j = 0; j < L.out; ++j) {
                            const float v = src[(size_t)i * L.out + j];
                            W[(size_t)i * L.out + j] = v;
                            Wt[(size_t)j * L.in_pad + i] = v;
                            if (fabsf(v) > L.wmax) L.wmax = fabsf(v);
                        }
                    src += (size_t)L.in * L.out;
                    for (int j = 0; j < L.out; ++j) b[j] = src[j];
                    src += L.out;
                    if (l == NNP_NLAYERS - 1) shift[s] += (double)b[0] / c->n_nets;
                    L.W = (float *)(W - blob.data()); L.Wt = (float *)(Wt - blob.data()); L.b = (float *)(b - blob.data());
                    if (c->tc_mode) { // tf32 hi / lo splits of both orientations (same rounding as the kernel's A split)
                        const size_t cnt = (size_t)L.in_pad * L.out;
                        float *dst[4] = {&blob[o], &blob[o + cnt], &blob[o + 2 * cnt], &blob[o + 3 * cnt]};
                        o += 4 * cnt;
                        const float *srcs[2] = {W, Wt};
                        for (int w = 0; w < 2; ++w)
                            for (size_t q = 0; q < cnt; ++q) {
                                uint32_t u; memcpy(&u, &srcs[w][q], 4);
                                uint32_t h = (u + 0x1000u) & 0xffffe000u;
                                float hf; memcpy(&hf, &h, 4);
                                float lf = srcs[w][q] - hf;
                                uint32_t lu; memcpy(&lu, &lf, 4);
                                lu = (lu + 0x1000u) & 0xffffe000u;
                                memcpy(&dst[2 * w][q], &h, 4);
                                memcpy(&dst[2 * w + 1][q], &lu, 4);
                            }
                        L.W_hi = (float *)(dst[0] - blob.data()); L.W_lo = (float *)(dst[1] - blob.data());
                        L.Wt_hi = (float *)(dst[2] - blob.data()); L.Wt_lo = (float *)(dst[3] - blob.data());
                    }
                }
    }
    int rc;
#define TRY(x) do { if ((rc = (x)) != NNP_OK) { g_create_error = c->err; nnp_destroy(c); return rc; } } while (0)
#define TRYCU(x) do { cudaError_t _e = (x); if (_e != cudaSuccess) { g_create_error = std::string(#x ": ") + cudaGetErrorString(_e); nnp_destroy(c); return _e == cudaErrorMemoryAllocation ? NNP_ENOMEM : NNP_ECUDA; } } while (0)
    TRY(dev_alloc(c, &c->d_params_blob, total));
    TRY(dev_alloc(c, &c->d_l1c_blob, total_l1c));
    TRY(dev_alloc(c, &c->d_fmap, (size_t)a.kpad));
    TRY(dev_alloc(c, &c->d_tri, (size_t)NNP_TRI_LEN));
    {
        std::vector<uint16_t> tri(NNP_TRI_LEN);
        nnp_aev_tri_table(tri.data());
        TRYCU(cudaMemcpy(c->d_tri, tri.data(), sizeof(uint16_t) * NNP_TRI_LEN, cudaMemcpyHostToDevice));
    }
    TRYCU(cudaMemcpy(c->d_params_blob, blob.data(), sizeof(float) * total, cudaMemcpyHostToDevice));
    for (size_t q = 0; q < (size_t)c->n_nets * S * NNP_NLAYERS; ++q) { // offsets -> device pointers
        LayerW &L = c->layers[q];
        L.W = c->d_params_blob + (size_t)L.W; L.Wt = c->d_params_blob + (size_t)L.Wt; L.b = c->d_params_blob + (size_t)L.b;
        if (c->tc_mode) {
            L.W_hi = c->d_params_blob + (size_t)L.W_hi; L.W_lo = c->d_params_blob + (size_t)L.W_lo;
            L.Wt_hi = c->d_params_blob + (size_t)L.Wt_hi; L.Wt_lo = c->d_params_blob + (size_t)L.Wt_lo;
        }
    }
    float imc[NNP_MAX_SPECIES] = {0}, ms[NNP_MAX_SPECIES] = {0}, es[NNP_MAX_SPECIES] = {0};
    for (int s = 0; s < S; ++s) {
        if (!(p->mass[s] > 0.f)) { g_create_error = "mass must be > 0"; nnp_destroy(c); return NNP_EINVAL; }
        c->mass[s] = ms[s] = p->mass[s];
        imc[s] = p->accel_conv / p->mass[s];
        c->e_shift[s] = es[s] = (float)(shift[s] + (p->self_energy ? (double)p->self_energy[s] : 0.0));
    }
    TRY(dev_alloc(c, &c->d_inv_mass_conv, NNP_MAX_SPECIES));
    TRY(dev_alloc(c, &c->d_mass, NNP_MAX_SPECIES));
    TRY(dev_alloc(c, &c->d_e_shift, NNP_MAX_SPECIES));
    TRY(dev_alloc(c, &c->d_lgv_c2, NNP_MAX_SPECIES));
    TRY(dev_alloc(c, &c->d_virial, 6));
    TRYCU(cudaMemcpy(c->d_inv_mass_conv, imc, sizeof(imc), cudaMemcpyHostToDevice));
    TRYCU(cudaMemcpy(c->d_mass, ms, sizeof(ms), cudaMemcpyHostToDevice));
    TRYCU(cudaMemcpy(c->d_e_shift, es, sizeof(es), cudaMemcpyHostToDevice));

    const size_t N = (size_t)max_atoms;
    TRY(dev_alloc(c, &c->pos, N)); TRY(dev_alloc(c, &c->pos_tmp, N));
    TRY(dev_alloc(c, &c->vel, N)); TRY(dev_alloc(c, &c->vel_tmp, N));
    TRY(dev_alloc(c, &c->frc, N)); TRY(dev_alloc(c, &c->xref, N));
    TRY(dev_alloc(c, &c->spc, N)); TRY(dev_alloc(c, &c->spc_tmp, N));
    TRY(dev_alloc(c, &c->orig, N)); TRY(dev_alloc(c, &c->orig_tmp, N));
    TRY(dev_alloc(c, &c->mol, N)); TRY(dev_alloc(c, &c->mol_tmp, N));
    TRY(dev_alloc(c, &c->mol_offsets, (size_t)max_mols + 1));
    TRY(dev_alloc(c, &c->key, N)); TRY(dev_alloc(c, &c->order, N));
    TRY(dev_alloc(c, &c->nbr_r, N * cap_r)); TRY(dev_alloc(c, &c->nbr_a, N * cap_a));
    TRY(dev_alloc(c, &c->seg_r, N * NNP_MAX_SPECIES)); TRY(dev_alloc(c, &c->seg_a, N * NNP_MAX_SPECIES));
    TRY(dev_alloc(c, &c->G, N * a.kpad));
    if (c->n_nets == 1) c->dG = c->G; // dE/dG overwrites G once layer 1 has consumed it
    else TRY(dev_alloc(c, &c->dG, N * a.kpad));
    for (int l = 0; l < 3; ++l) TRY(dev_alloc(c, &c->H[l], N * c->hmax[l] * (size_t)c->n_nets));
    TRY(dev_alloc(c, &c->e_atom, N));
    TRY(dev_alloc(c, &c->e_mol, (size_t)max_mols));
    TRY(dev_alloc(c, &c->ekin, (size_t)max_mols));
    TRY(dev_alloc(c, &c->flags, 16));
    TRY(dev_alloc(c, &c->io_xyz, 3 * N)); TRY(dev_alloc(c, &c->io_vel, 3 * N)); TRY(dev_alloc(c, &c->io_species, N));
    TRY(dev_alloc(c, &c->d_res, 8));
    if (cudaHostAlloc((void **)&c->h_res, 8 * sizeof(double), cudaHostAllocDefault) != cudaSuccess) { c->h_res = nullptr; cudaGetLastError(); }
    TRYCU(cudaMemset(c->flags, 0, sizeof(int) * 16));
    TRY(dev_alloc(c, &c->aev_sched, 2 * NNP_AEV_SCHED_LEN));
    TRYCU(cudaMemset(c->aev_sched, 0, sizeof(int) * 2 * NNP_AEV_SCHED_LEN));
    TRYCU(cudaMemset(c->ekin, 0, sizeof(double) * (size_t)max_mols));
    TRYCU(cudaDeviceSynchronize());
#undef TRY
#undef TRYCU
    *out = c;
    return NNP_OK;
}

// cells narrower than this are replicated into the smallest supercell that reaches it (nnp_set_system_cell)
static const float kPbcSkinReserve = 0.5f;

static int set_system_impl(nnp_ctx *c, int n_atoms, const int32_t *d_species, const float *d_xyz, const float cell[9],
                           int n_mols, const int32_t *d_mol_offsets)
{
    if (n_atoms > 0 && (!d_species || !d_xyz)) NNP_FAIL(c, NNP_EINVAL, "null argument");
    if (n_atoms < 0 || n_atoms > c->max_atoms) NNP_FAIL(c, NNP_EINVAL, "n_atoms %d outside [0, max_atoms=%d]", n_atoms, c->max_atoms);
    if (!d_mol_offsets) n_mols = 1;
    if (n_mols < 1 || n_mols > c->max_mols) NNP_FAIL(c, NNP_EINVAL, "n_mols %d outside [1, max_mols=%d]", n_mols, c->max_mols);
    bool any = false;
    for (int q = 0; q < 9; ++q) any = any || cell[q] != 0.f;
    int periodic = 0, tric = 0, m[3] = {1, 1, 1};
    if (any) {
        double h[9], rec[9];
        for (int q = 0; q < 9; ++q) h[q] = cell[q];
        cross3f(h + 3, h + 6, rec); cross3f(h + 6, h, rec + 3); cross3f(h, h + 3, rec + 6);
        const double vol = h[0] * rec[0] + h[1] * rec[1] + h[2] * rec[2];
        if (!(fabs(vol) > 1e-12)) NNP_FAIL(c, NNP_EINVAL, "cell vectors must be all zero (non-periodic) or span a volume");
        periodic = 1;
        tric = cell[1] != 0.f || cell[2] != 0.f || cell[3] != 0.f || cell[5] != 0.f || cell[6] != 0.f || cell[7] != 0.f;
        if (!tric && (cell[0] <= 0.f || cell[4] <= 0.f || cell[8] <= 0.f)) NNP_FAIL(c, NNP_EINVAL, "box edges must be positive");
        const double need = 2.0 * ((double)c->aev.rcr + (double)kPbcSkinReserve);
        for (int d = 0; d < 3; ++d) {
            const double w = fabs(vol) / sqrt(rec[3 * d] * rec[3 * d] + rec[3 * d + 1] * rec[3 * d + 1] + rec[3 * d + 2] * rec[3 * d + 2]);
            if (w < need) m[d] = (int)ceil(need / w - 1e-9);
        }
    }
    const long rep = (long)m[0] * m[1] * m[2];
    if (rep > 1) {
        if (n_mols != 1) NNP_FAIL(c, NNP_EBOX, "a batch of cells narrower than 2 (rcr + 0.5 A) is not supported");
        if ((long)n_atoms * rep > c->max_atoms)
            NNP_FAIL(c, NNP_EBOX, "cell narrower than 2 (rcr + 0.5 A): all periodic images are evaluated on a %d x %d x %d supercell, "
                     "which needs max_atoms >= %ld", m[0], m[1], m[2], (long)n_atoms * rep);
    }
    CU(c, cudaSetDevice(c->device));
    c->n_user = n_atoms; c->rep = (int)rep; c->n = n_atoms * (int)rep; c->n_mols = n_mols; c->periodic = periodic; c->tric = tric;
    for (int d = 0; d < 3; ++d) {
        c->rep_m[d] = m[d];
        for (int q = 0; q < 3; ++q) { c->cell_user[3 * d + q] = cell[3 * d + q]; c->cell[3 * d + q] = (float)m[d] * cell[3 * d + q]; }
        c->box[d] = c->cell[4 * d];
    }
    c->have_system = 1; c->have_lists = 0; c->have_forces = 0; c->md_ready = 0;
    drop_md_graph(c);
    int *bins = c->flags + 8; // [8..15] species histogram, [3] bad-species marker
    CU(c, cudaMemsetAsync(c->flags, 0, sizeof(int) * 16, c->stream));
    int h_counts[NNP_MAX_SPECIES] = {0};
    if (n_atoms > 0) {
        if (d_mol_offsets)
            CU(c, cudaMemcpyAsync(c->mol_offsets, d_mol_offsets, sizeof(int) * (n_mols + 1), cudaMemcpyDeviceToDevice, c->stream));
        RepInfo ri;
        ri.n_user = n_atoms;
        for (int d = 0; d < 3; ++d) ri.m[d] = m[d];
        for (int q = 0; q < 9; ++q) ri.cu[q] = cell[q];
        k_init_system<<<nnp_div_up(c->n, T), T, 0, c->stream>>>(c->n, d_species, d_xyz, d_mol_offsets ? c->mol_offsets : nullptr,
                                                                n_mols, c->pos, c->vel, c->spc, c->orig, c->mol, bins, c->S,
                                                                c->flags + 3, ri);
        c->launches += 1;
        int bad = 0;
        CU(c, cudaMemcpyAsync(h_counts, bins, sizeof(int) * NNP_MAX_SPECIES, cudaMemcpyDeviceToHost, c->stream));
        CU(c, cudaMemcpyAsync(&bad, c->flags + 3, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
        CU(c, cudaStreamSynchronize(c->stream));
        if (bad) {
            c->have_system = 0;
            NNP_FAIL(c, NNP_EINVAL, (bad & 1) ? "species index outside [0, n_species)"
                                              : "mol_offsets must be 0 = o[0] <= o[1] <= ... <= o[n_mols] = n_atoms");
        }
    }
    c->bucket_off[0] = 0;
    for (int s = 0; s < NNP_MAX_SPECIES; ++s) c->bucket_off[s + 1] = c->bucket_off[s] + (s < c->S ? h_counts[s] : 0);
    unsigned mask = 0;
    for (int s = 0; s < c->S; ++s)
        if (h_counts[s] > 0) mask |= 1u << s;
    if (c->dense_aev || mask == 0) mask = (1u << c->S) - 1u;
    int rc = set_layout(c, mask);
    if (rc) return rc;
    return nnp_fused_setup(c);
}

int nnp_set_system(nnp_ctx *c, int n_atoms, const int32_t *d_species, const float *d_xyz, const float h_box[3],
                   int n_mols, const int32_t *d_mol_offsets)
{
    if (!c) return NNP_EINVAL;
    float cell[9] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    if (h_box) {
        const int nper = (h_box[0] > 0.f) + (h_box[1] > 0.f) + (h_box[2] > 0.f);
        if (nper != 0 && nper != 3) NNP_FAIL(c, NNP_EINVAL, "box must be all zero (non-periodic) or all positive");
        cell[0] = h_box[0]; cell[4] = h_box[1]; cell[8] = h_box[2];
    }
    return set_system_impl(c, n_atoms, d_species, d_xyz, cell, n_mols, d_mol_offsets);
}

int nnp_set_system_cell(nnp_ctx *c, int n_atoms, const int32_t *d_species, const float *d_xyz, const float h_cell[9],
                        int n_mols, const int32_t *d_mol_offsets)
{
    if (!c) return NNP_EINVAL;
    static const float zero[9] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    return set_system_impl(c, n_atoms, d_species, d_xyz, h_cell ? h_cell : zero, n_mols, d_mol_offsets);
}

int nnp_set_positions(nnp_ctx *c, const float *d_xyz)
{
    if (!c) return NNP_EINVAL;
    if (!c->have_system || !d_xyz) NNP_FAIL(c, NNP_EINVAL, "no system loaded / null argument");
    if (c->n == 0) return NNP_OK;
    if (c->rep > 1) {
        RepInfo rep;
        rep.n_user = c->n_user;
        for (int d = 0; d < 3; ++d) rep.m[d] = c->rep_m[d];
        for (int q = 0; q < 9; ++q) rep.cu[q] = c->cell_user[q];
        k_set_positions_rep<<<nnp_div_up(c->n, T), T, 0, c->stream>>>(c->n, d_xyz, c->orig, c->pos, rep);
        c->launches += 1;
    } else {
        nnp_launch_permute_in3(c, d_xyz, c->pos);
    }
    c->have_forces = 0;
    return NNP_OK;
}

int nnp_build_neighbors(nnp_ctx *c, float skin)
{
    if (!c) return NNP_EINVAL;
    if (!c->have_system) NNP_FAIL(c, NNP_ESTALE, "nnp_set_system first");
    if (!(skin >= 0.f)) NNP_FAIL(c, NNP_EINVAL, "skin must be >= 0");
    CU(c, cudaSetDevice(c->device));
    // A captured MD-step graph has the skin, the grid and the key-array pointers baked into its kernel arguments:
    // it is re-captured by the next nnp_md_step.
    drop_md_graph(c);
    c->skin = skin;
    int rc = setup_grid(c, skin);
    if (rc) return rc;
    if (c->n > 0) nnp_launch_build(c, nullptr);
    CU(c, cudaGetLastError());
    c->have_lists = 1;
    c->have_forces = 0;
    return NNP_OK;
}

int nnp_get_neighbors(nnp_ctx *c, int which, int32_t *d_counts, int32_t *d_list, int stride)
{
    if (!c) return NNP_EINVAL;
    if (!c->have_lists) NNP_FAIL(c, NNP_ESTALE, "no neighbour list");
    if (!d_counts || !d_list || stride < 1 || (which != 0 && which != 1)) NNP_FAIL(c, NNP_EINVAL, "bad argument");
    if (c->n > 0) {
        k_get_neighbors<<<nnp_div_up(c->n, T), T, 0, c->stream>>>(c->n, which ? c->nbr_a : c->nbr_r, which ? c->seg_a : c->seg_r,
                                                                 which ? c->aev.cap_a : c->aev.cap_r, c->orig, c->n_user, d_counts, d_list, stride);
        c->launches += 1;
    }
    return check_flags(c);
}

static int energy_forces_impl(nnp_ctx *c, double *d_energy /* nullptr: leave in e_mol */, float *d_forces)
{
    if (!c->have_lists) NNP_FAIL(c, NNP_ESTALE, "nnp_build_neighbors first");
    CU(c, cudaSetDevice(c->device));
    if (c->n == 0) {
        CU(c, cudaMemsetAsync(c->e_mol, 0, sizeof(double) * c->n_mols, c->stream));
    } else {
        prof_begin(c);
        int rc = run_forces(c);
        c->prof_active = 0;
        if (rc) return rc;
        if (d_forces) nnp_launch_unpermute3(c, c->frc, d_forces);
    }
    if (d_energy) CU(c, cudaMemcpyAsync(d_energy, c->e_mol, sizeof(double) * c->n_mols, cudaMemcpyDeviceToDevice, c->stream));
    return NNP_OK;
}

int nnp_energy_forces(nnp_ctx *c, double *d_energy, float *d_forces)
{
    if (!c) return NNP_EINVAL;
    if (!d_energy) NNP_FAIL(c, NNP_EINVAL, "null energy pointer");
    return energy_forces_impl(c, d_energy, d_forces);
}

// symmetric 3x3 from the six sums xx yy zz xy xz yz of the reverse AEV kernel
__global__ void k_expand_virial(const double *__restrict__ v6, double scale, double *__restrict__ v9)
{
    const int map[9] = {0, 3, 4, 3, 1, 5, 4, 5, 2};
    if (threadIdx.x < 9) v9[threadIdx.x] = v6[map[threadIdx.x]] * scale;
}

int nnp_energy_forces_virial(nnp_ctx *c, double *d_energy, float *d_forces, double *d_virial)
{
    if (!c) return NNP_EINVAL;
    if (!d_energy || !d_virial) NNP_FAIL(c, NNP_EINVAL, "null energy / virial pointer");
    if (c->n_mols != 1) NNP_FAIL(c, NNP_EINVAL, "the virial is defined for one structure (n_mols = 1)");
    CU(c, cudaSetDevice(c->device));
    CU(c, cudaMemsetAsync(c->d_virial, 0, sizeof(double) * 6, c->stream));
    c->want_virial = 1;
    const int rc = energy_forces_impl(c, d_energy, d_forces);
    c->want_virial = 0;
    if (rc) return rc;
    k_expand_virial<<<1, 32, 0, c->stream>>>(c->d_virial, 1.0 / (double)c->rep, d_virial);
    c->launches += 1;
    CU(c, cudaGetLastError());
    return NNP_OK;
}

int nnp_get_aev(nnp_ctx *c, float *d_aev)
{
    if (!c) return NNP_EINVAL;
    if (!c->have_lists || !d_aev) NNP_FAIL(c, NNP_ESTALE, "no neighbour list / null argument");
    if (c->n == 0) return NNP_OK;
    nnp_launch_aev_forward(c); // G may have been overwritten by dE/dG: recompute
    k_get_aev<<<c->n, 128, 0, c->stream>>>(c->n, c->aev_len_full, c->aev.aev_len, c->aev.kpad, c->G, c->d_fmap, c->orig, c->n_user, d_aev);
    c->launches += 1;
    c->have_forces = 0;
    CU(c, cudaGetLastError());
    return NNP_OK;
}

int nnp_get_atomic_energies(nnp_ctx *c, float *d_e_atom)
{
    if (!c) return NNP_EINVAL;
    if (!c->have_forces || !d_e_atom) NNP_FAIL(c, NNP_ESTALE, "nnp_energy_forces first / null argument");
    k_get_e_atom<<<nnp_div_up(c->n, T), T, 0, c->stream>>>(c->n, c->e_atom, c->spc, c->d_e_shift, 1.0f / c->n_nets, c->orig, c->n_user, d_e_atom);
    c->launches += 1;
    return NNP_OK;
}

int nnp_md_init(nnp_ctx *c, const float *d_vel, float dt_fs, float skin)
{
    if (!c) return NNP_EINVAL;
    if (!c->have_system) NNP_FAIL(c, NNP_ESTALE, "nnp_set_system first");
    if (!d_vel || !(dt_fs > 0.f) || !(skin > 0.f)) NNP_FAIL(c, NNP_EINVAL, "need velocities, dt > 0, skin > 0");
    if (c->n == 0) NNP_FAIL(c, NNP_EINVAL, "empty system");
    CU(c, cudaSetDevice(c->device));
    if (c->rep > 1 && c->rep_stage_cap < 2 * c->n_user) { // a replicated small cell: staging for the state of copy 0
        CU(c, cudaStreamSynchronize(c->stream));
        dev_free(c, c->rep_stage);
        c->rep_stage = nullptr;
        c->rep_stage_cap = 0;
        int rc0 = dev_alloc(c, &c->rep_stage, (size_t)2 * c->n_user);
        if (rc0) return rc0;
        c->rep_stage_cap = 2 * c->n_user;
    }
    nnp_launch_permute_in3(c, d_vel, c->vel);
    c->dt = dt_fs;
    c->lgv_gamma = 0.f; // velocity Verlet until nnp_md_set_langevin
    drop_md_graph(c);
    CU(c, cudaMemsetAsync(c->flags + 1, 0, sizeof(int) * 4, c->stream)); // rebuild request and counter, Langevin step counter
    int rc = nnp_build_neighbors(c, skin);
    if (rc) return rc;
    // the initial build counts as rebuild 1 (k_finish_build)
    rc = run_forces(c);
    if (rc) return rc;
    const float dt = c->dt;
    c->dt = 0.f;
    nnp_launch_kick_ke(c, 0); // kinetic energy of the initial velocities
    c->dt = dt;
    c->md_ready = 1;
    return NNP_OK;
}

int nnp_md_set_langevin(nnp_ctx *c, float gamma, float kT, uint64_t seed)
{
    if (!c) return NNP_EINVAL;
    if (!(gamma >= 0.f) || !(kT >= 0.f)) NNP_FAIL(c, NNP_EINVAL, "gamma and kT must be >= 0");
    if (!c->md_ready) NNP_FAIL(c, NNP_ESTALE, "nnp_md_init first");
    CU(c, cudaSetDevice(c->device));
    c->lgv_gamma = gamma; c->lgv_kT = kT; c->lgv_seed = seed;
    const double c1 = exp(-(double)gamma * (double)c->dt);
    c->lgv_c1 = (float)c1;
    float c2[NNP_MAX_SPECIES] = {0};
    for (int s = 0; s < c->S; ++s) c2[s] = (float)sqrt((1.0 - c1 * c1) * (double)kT * (double)c->accel_conv / (double)c->mass[s]);
    CU(c, cudaMemcpyAsync(c->d_lgv_c2, c2, sizeof(c2), cudaMemcpyHostToDevice, c->stream));
    CU(c, cudaStreamSynchronize(c->stream)); // c2 is a stack array
    drop_md_graph(c);                        // the drift kernel and its constants are baked into the graph
    return NNP_OK;
}

int nnp_md_step(nnp_ctx *c, int n_steps)
{
    if (!c) return NNP_EINVAL;
    if (!c->md_ready) NNP_FAIL(c, NNP_ESTALE, "nnp_md_init first");
    if (n_steps < 0) NNP_FAIL(c, NNP_EINVAL, "n_steps < 0");
    CU(c, cudaSetDevice(c->device));
    if (!c->no_graph && !c->md_exec && n_steps > 0) {
        int rc = build_md_graph(c);
        if (rc) return rc;
    }
    for (int step = 0; step < n_steps; ++step) {
        prof_begin(c);
        if (c->md_exec && !c->prof_active) { // the per-stage event marks need the kernel-by-kernel path
            CU(c, cudaGraphLaunch(c->md_exec, c->stream));
            c->launches += c->md_graph_launches;
            continue;
        }
        nnp_launch_kick_drift(c);
        nnp_prof_mark(c, 0);
        nnp_launch_build(c, c->flags + 1); // every kernel returns at once unless the drift requested a rebuild
        nnp_prof_mark(c, 1);
        int rc = run_forces(c);
        if (rc) { c->prof_active = 0; return rc; }
        nnp_launch_kick_ke(c, 1);
        nnp_prof_mark(c, 11);
        c->prof_active = 0;
    }
    return NNP_OK;
}

int nnp_get_state(nnp_ctx *c, float *d_xyz, float *d_vel, double *d_epot, double *d_ekin, int32_t *d_n_rebuilds)
{
    if (!c) return NNP_EINVAL;
    if (!c->have_system) NNP_FAIL(c, NNP_ESTALE, "no system");
    if (c->n > 0) {
        if (d_xyz) nnp_launch_unpermute3(c, c->pos, d_xyz);
        if (d_vel) nnp_launch_unpermute3(c, c->vel, d_vel);
    }
    if (d_epot) CU(c, cudaMemcpyAsync(d_epot, c->e_mol, sizeof(double) * c->n_mols, cudaMemcpyDeviceToDevice, c->stream));
    if (d_ekin) CU(c, cudaMemcpyAsync(d_ekin, c->ekin, sizeof(double) * c->n_mols, cudaMemcpyDeviceToDevice, c->stream));
    if (d_n_rebuilds) CU(c, cudaMemcpyAsync(d_n_rebuilds, c->flags + 2, sizeof(int), cudaMemcpyDeviceToDevice, c->stream));
    return NNP_OK;
}

int nnp_profile(nnp_ctx *c, int stride)
{
    if (!c || stride < 0) return NNP_EINVAL;
    prof_collect(c);
    c->prof_stride = stride;
    c->prof_calls = 0;
    if (stride == 0)
        for (int k = 0; k < NNP_N_STAGES; ++k) { c->prof_ms[k] = 0.0; c->prof_n[k] = 0; }
    return NNP_OK;
}

int nnp_profile_read(nnp_ctx *c, double *h_ms_sum, int64_t *h_samples)
{
    if (!c || !h_ms_sum || !h_samples) return NNP_EINVAL;
    prof_collect(c);
    for (int k = 0; k < NNP_N_STAGES; ++k) { h_ms_sum[k] = c->prof_ms[k]; h_samples[k] = c->prof_n[k]; }
    return NNP_OK;
}

int nnp_sync(nnp_ctx *c)
{
    if (!c) return NNP_EINVAL;
    CU(c, cudaSetDevice(c->device));
    return check_flags(c);
}

int nnp_energy_forces_host(nnp_ctx *c, int n_atoms, const int32_t *h_species, const float *h_xyz, const float h_box[3],
                           int n_mols, const int32_t *h_mol_offsets, float skin, double *h_energy, float *h_forces)
{
    if (!c) return NNP_EINVAL;
    if ((n_atoms > 0 && (!h_species || !h_xyz)) || !h_energy) NNP_FAIL(c, NNP_EINVAL, "null argument");
    if (n_atoms < 0 || n_atoms > c->max_atoms) NNP_FAIL(c, NNP_EINVAL, "n_atoms outside [0, max_atoms]");
    if (h_mol_offsets && (n_mols < 1 || n_mols > c->max_mols)) NNP_FAIL(c, NNP_EINVAL, "n_mols outside [1, max_mols]");
    CU(c, cudaSetDevice(c->device));
    CU(c, cudaMemcpyAsync(c->io_species, h_species, sizeof(int) * (size_t)n_atoms, cudaMemcpyHostToDevice, c->stream));
    CU(c, cudaMemcpyAsync(c->io_xyz, h_xyz, sizeof(float) * 3 * (size_t)n_atoms, cudaMemcpyHostToDevice, c->stream));
    int *d_off = nullptr;
    if (h_mol_offsets) {
        d_off = c->key; // scratch until the build; set_system copies it into mol_offsets
        if (n_mols + 1 > c->max_atoms) NNP_FAIL(c, NNP_EINVAL, "n_mols + 1 > max_atoms");
        CU(c, cudaMemcpyAsync(d_off, h_mol_offsets, sizeof(int) * (n_mols + 1), cudaMemcpyHostToDevice, c->stream));
    }
    int rc = nnp_set_system(c, n_atoms, c->io_species, c->io_xyz, h_box, n_mols, d_off);
    if (rc) return rc;
    if ((rc = nnp_build_neighbors(c, skin))) return rc;
    // energies stay in e_mol; forces go through io_vel as staging
    if ((rc = energy_forces_impl(c, nullptr, h_forces ? c->io_vel : nullptr))) return rc;
    CU(c, cudaMemcpyAsync(h_energy, c->e_mol, sizeof(double) * c->n_mols, cudaMemcpyDeviceToHost, c->stream));
    if (h_forces && n_atoms > 0)
        CU(c, cudaMemcpyAsync(h_forces, c->io_vel, sizeof(float) * 3 * (size_t)n_atoms, cudaMemcpyDeviceToHost, c->stream));
    return check_flags(c);
}

int nnp_md_step_host(nnp_ctx *c, float *h_xyz, float *h_vel, int n_steps, double *h_epot, double *h_ekin)
{
    if (!c) return NNP_EINVAL;
    if (!c->md_ready) NNP_FAIL(c, NNP_ESTALE, "nnp_md_init first");
    if (!h_xyz || !h_vel) NNP_FAIL(c, NNP_EINVAL, "null argument");
    if (c->n_mols != 1) NNP_FAIL(c, NNP_EINVAL, "nnp_md_step_host returns the energies of one structure: use nnp_md_step / nnp_get_state for a batch");
    CU(c, cudaSetDevice(c->device));
    const size_t bytes = sizeof(float) * 3 * (size_t)c->n;
    CU(c, cudaMemcpyAsync(c->io_xyz, h_xyz, bytes, cudaMemcpyHostToDevice, c->stream));
    CU(c, cudaMemcpyAsync(c->io_vel, h_vel, bytes, cudaMemcpyHostToDevice, c->stream));
    nnp_launch_permute_in3x2(c, c->io_xyz, c->pos, c->io_vel, c->vel);
    nnp_launch_sync_copies(c, 0); // (a replicated small cell: the copies get their lattice shifts back)
    int rc = nnp_md_step(c, n_steps);
    if (rc) return rc;
    nnp_launch_unpermute3x2(c, c->pos, c->io_xyz, c->vel, c->io_vel);
    CU(c, cudaMemcpyAsync(h_xyz, c->io_xyz, bytes, cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaMemcpyAsync(h_vel, c->io_vel, bytes, cudaMemcpyDeviceToHost, c->stream));
    if (!c->h_res) { // no pinned staging: one copy per scalar
        if (h_epot) CU(c, cudaMemcpyAsync(h_epot, c->e_mol, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        if (h_ekin) CU(c, cudaMemcpyAsync(h_ekin, c->ekin, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        return check_flags(c);
    }
    // energies and the device-side error flags come back in ONE pinned copy (three pageable 8-12 byte copies before)
    nnp_launch_pack_result(c);
    CU(c, cudaMemcpyAsync(c->h_res, c->d_res, 5 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CU(c, cudaStreamSynchronize(c->stream));
    if (h_epot) *h_epot = c->h_res[0];
    if (h_ekin) *h_ekin = c->h_res[1];
    const int f0 = (int)c->h_res[2];
    if (f0 & (NNP_FLAG_CAP_R | NNP_FLAG_CAP_A))
        NNP_FAIL(c, NNP_ECAPACITY, "neighbour capacity exceeded (%s): recreate with larger cap_r/cap_a",
                 (f0 & NNP_FLAG_CAP_R) ? "radial" : "angular");
    if (f0 & NNP_FLAG_RANGE)
        NNP_FAIL(c, NNP_ERANGE, "mm_mode 4: an activation exceeded the range of the scaled fp16 split; use mm_mode 1");
    return NNP_OK;
}

} // extern "C"
