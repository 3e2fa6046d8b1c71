/*
 * nnp_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of what the ANI-2x energy/force/MD hot path computes
 * (FeNNol paper, arxiv 2405.01491, /root/reference/PAPER.md; Fig. 2, SecII.A,
 * SecII.B, SecV, Eq. (A9)/L443 for the angular symmetry function).  The paper never
 * prints the ANI equations or constants, so the step-by-step definition followed here is
 * SURVEY.md Sec.8(c) C1 (O1..O7) with the readings of Sec.8(c) C2 -- each function cites its item.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
 * load this file.  It shares no code, header, table or helper with the CUDA path under
 * paper_2405_01491_b200/csrc/.  There is no blocking, fusion or reordering beyond what the
 * definition states: neighbours by brute force (or an independent, separately tested uniform
 * grid for large N), direct sums for the AEV, a textbook MLP, an analytic gradient that the
 * tests pin with central finite differences.
 *
 * Parity pins (tests/test_oracle_*.py): AEV length closed form, hand-evaluated dimer/trimer
 * values, MLP vs numpy matmul, finite differences, net force / net torque zero, translation,
 * rotation, lattice-shift, wrap and same-species permutation invariance, cutoff continuity,
 * box replication extensivity, ensemble and batch identities, velocity-Verlet reversibility
 * and dt^2 energy error.  Absolute values against the paper: "parity unpinned" (the paper
 * prints none for this path; SURVEY.md Sec.8(c) C3 last row).
 *
 * Build:  gcc -O2 -std=c99 -ffp-contract=off -fopenmp -shared -fPIC nnp_oracle.c -lm
 * Units: kcal/mol, Angstrom, fs, amu (reading B6).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

typedef struct {
    int n_species;          /* S = 7 for ANI-2x (H,C,N,O,S,F,Cl = 0..6, reading B2) */
    double rcr, rca;        /* radial / angular cutoff (5.1 / 3.5 A, reading A1) */
    double eta_r;           /* radial Gaussian width */
    int n_shf_r;            /* 16 */
    const double *shf_r;
    double eta_a, zeta;     /* angular */
    int n_shf_a;            /* 8 */
    const double *shf_a;
    int n_shf_z;            /* 4 */
    const double *shf_z;
    double celu_alpha;      /* 0.1 */
    int n_nets;             /* 1 or 8 (reading B5: arithmetic mean) */
    int n_layers;           /* affine layers per network (4) */
    const int *widths;      /* [S][n_layers+1] */
    const double *params;   /* flat: for net, for species, for layer: W[in][out] row-major, then b[out] */
    const double *self_energy; /* [S] or NULL (reading B4) */
} orc_model;

/* ---- closed-form sizes (SURVEY 8(c) C3 "AEV length") ------------------------------------- */
int orc_n_pairs(int S) { return S * (S + 1) / 2; }
int orc_aev_len(const orc_model *m)
{
    return m->n_species * m->n_shf_r + orc_n_pairs(m->n_species) * m->n_shf_a * m->n_shf_z;
}
/* O3: p(s,t), s<=t, row-major upper triangle: row s starts at sum_{u<s}(S-u). */
int orc_pair_index(int S, int s, int t)
{
    if (s > t) { int u = s; s = t; t = u; }
    return s * (2 * S + 1 - s) / 2 + (t - s);
}
long orc_params_per_net(const orc_model *m)
{
    long tot = 0;
    for (int s = 0; s < m->n_species; ++s)
        for (int l = 0; l < m->n_layers; ++l) {
            long in = m->widths[s * (m->n_layers + 1) + l], out = m->widths[s * (m->n_layers + 1) + l + 1];
            tot += in * out + out;
        }
    return tot;
}
static const double *layer_ptr(const orc_model *m, int net, int s, int l)
{
    long off = net * orc_params_per_net(m);
    for (int u = 0; u < m->n_species; ++u)
        for (int k = 0; k < m->n_layers; ++k) {
            if (u == s && k == l) return m->params + off;
            long in = m->widths[u * (m->n_layers + 1) + k], out = m->widths[u * (m->n_layers + 1) + k + 1];
            off += in * out + out;
        }
    return NULL;
}

/* ---- O1: neighbours ---------------------------------------------------------------------- */
/* fp64 minimum-image displacement d = x_j - x_i (reading C1: cubic/orthorhombic box, min image). */
static void disp(const double *xi, const double *xj, const double *box, double d[3])
{
    for (int c = 0; c < 3; ++c) {
        d[c] = xj[c] - xi[c];
        if (box && box[c] > 0.0) d[c] -= box[c] * round(d[c] / box[c]);
    }
}

/* Reading A3: the DEFINED list-membership predicate is fp32 with a fixed operation order:
 *   dx = xj - xi (rn); dx = dx - L*rintf(dx*invL) (separate rn mul, rn mul, rn sub; invL = 1.0f/L);
 *   r2 = (dx*dx + dy*dy) + dz*dz (each op rn, no FMA); member iff r2 < rlist*rlist (rn product).
 * This file is compiled with -ffp-contract=off so no operation below is fused. */
static int within_f32(const float *xi, const float *xj, const float *L, const float *invL, float rl2)
{
    float d[3];
    for (int c = 0; c < 3; ++c) {
        float t = xj[c] - xi[c];
        if (L[c] > 0.0f) {
            float q = t * invL[c];
            float k = rintf(q);
            float s = L[c] * k;
            t = t - s;
        }
        d[c] = t;
    }
    float a = d[0] * d[0];
    float b = d[1] * d[1];
    float c2 = d[2] * d[2];
    float r2 = (a + b) + c2;
    return r2 < rl2;
}

/* Brute force O(N^2): directed list (each pair twice); same molecule only.
 * fp32_pred=0: fp64 r2 < rcut^2; fp32_pred=1: reading A3 with rlist = (float)rcut.
 * Returns max row length, or -(needed) if some row exceeds cap (list then truncated). */
int orc_neighbors_brute(int n, const double *xyz, const double *box, const int *mol_id, double rcut,
                        int fp32_pred, int cap, int *counts, int *list)
{
    float Lf[3] = {0, 0, 0}, invL[3] = {0, 0, 0};
    if (box) for (int c = 0; c < 3; ++c) { Lf[c] = (float)box[c]; invL[c] = Lf[c] > 0 ? 1.0f / Lf[c] : 0.0f; }
    float rl = (float)rcut;
    float rl2 = rl * rl;
    int maxc = 0;
#pragma omp parallel for schedule(dynamic, 64) reduction(max : maxc)
    for (int i = 0; i < n; ++i) {
        int c = 0;
        float xi[3] = {(float)xyz[3 * i], (float)xyz[3 * i + 1], (float)xyz[3 * i + 2]};
        for (int j = 0; j < n; ++j) {
            if (j == i) continue;
            if (mol_id && mol_id[i] != mol_id[j]) continue;
            int in;
            if (fp32_pred) {
                float xj[3] = {(float)xyz[3 * j], (float)xyz[3 * j + 1], (float)xyz[3 * j + 2]};
                in = within_f32(xi, xj, Lf, invL, rl2);
            } else {
                double d[3];
                disp(xyz + 3 * i, xyz + 3 * j, box, d);
                in = (d[0] * d[0] + d[1] * d[1] + d[2] * d[2]) < rcut * rcut;
            }
            if (in) { if (c < cap) list[(long)i * cap + c] = j; ++c; }
        }
        counts[i] = c;
        if (c > maxc) maxc = c;
    }
    return maxc > cap ? -maxc : maxc;
}

/* ---- NEXT-2 (second part; "optionally cell vectors", L49 shift vectors, L307
 * "minimum image or all images"): a GENERAL cell (rows of cell[9] are the lattice vectors a, b, c; triclinic allowed) with
 * ALL periodic images, written out as the definition: atom i sees every image x_j + s_0 a + s_1 b + s_2 c (s integer, the
 * pair (j = i, s = 0) excluded) closer than rcut - including images of itself and several images of the same atom when the
 * cell is smaller than 2 rcut.  A list entry is (j, s).  For cells wider than 2 rcut this is the minimum-image list. */
static void disp_cell(const double *xi, const double *xj, const double *cell, const int *s, double d[3])
{
    for (int c = 0; c < 3; ++c)
        d[c] = xj[c] - xi[c] + (double)s[0] * cell[c] + (double)s[1] * cell[3 + c] + (double)s[2] * cell[6 + c];
}

static void cross3(const double *a, const double *b, double *o)
{
    o[0] = a[1] * b[2] - a[2] * b[1]; o[1] = a[2] * b[0] - a[0] * b[2]; o[2] = a[0] * b[1] - a[1] * b[0];
}

/* Brute force over pairs and shifts, fp64 predicate r2 < rcut^2.  The shifts that can matter: a vector shorter than rcut
 * has |fractional component c| <= rcut / w_c, w_c = volume / |area of the face spanned by the other two vectors| (the
 * perpendicular width); every integer s_c with |frac_c(x_j - x_i) + s_c| <= rcut / w_c is tried.
 * counts[n], list[n][cap], shifts[n][cap][3].  Returns max row length, or -(needed) if some row exceeds cap. */
int orc_neighbors_cell(int n, const double *xyz, const double *cell, const int *mol_id, double rcut, int cap,
                       int *counts, int *list, int *shifts)
{
    double rec[9], vol, reach[3]; /* rec rows: reciprocal vectors b x c, c x a, a x b (frac_c = rec_c . x / vol) */
    cross3(cell + 3, cell + 6, rec); cross3(cell + 6, cell, rec + 3); cross3(cell, cell + 3, rec + 6);
    vol = cell[0] * rec[0] + cell[1] * rec[1] + cell[2] * rec[2];
    if (!(fabs(vol) > 0.0)) return -1000000000;
    for (int c = 0; c < 3; ++c) {
        double area = sqrt(rec[3 * c] * rec[3 * c] + rec[3 * c + 1] * rec[3 * c + 1] + rec[3 * c + 2] * rec[3 * c + 2]);
        reach[c] = rcut * area / fabs(vol); /* rcut / w_c */
    }
    int maxc = 0;
#pragma omp parallel for schedule(dynamic, 16) reduction(max : maxc)
    for (int i = 0; i < n; ++i) {
        int cnt = 0;
        for (int j = 0; j < n; ++j) {
            if (mol_id && mol_id[i] != mol_id[j]) continue;
            double f[3];
            for (int c = 0; c < 3; ++c) {
                double t = 0.0;
                for (int q = 0; q < 3; ++q) t += rec[3 * c + q] * (xyz[3 * j + q] - xyz[3 * i + q]);
                f[c] = t / vol;
            }
            int lo[3], hi[3];
            for (int c = 0; c < 3; ++c) { lo[c] = (int)ceil(-reach[c] - f[c] - 1e-9); hi[c] = (int)floor(reach[c] - f[c] + 1e-9); }
            for (int s0 = lo[0]; s0 <= hi[0]; ++s0)
                for (int s1 = lo[1]; s1 <= hi[1]; ++s1)
                    for (int s2 = lo[2]; s2 <= hi[2]; ++s2) {
                        if (j == i && s0 == 0 && s1 == 0 && s2 == 0) continue;
                        int sh[3] = {s0, s1, s2};
                        double d[3];
                        disp_cell(xyz + 3 * i, xyz + 3 * j, cell, sh, d);
                        if ((d[0] * d[0] + d[1] * d[1] + d[2] * d[2]) < rcut * rcut) {
                            if (cnt < cap) {
                                list[(long)i * cap + cnt] = j;
                                shifts[((long)i * cap + cnt) * 3] = s0;
                                shifts[((long)i * cap + cnt) * 3 + 1] = s1;
                                shifts[((long)i * cap + cnt) * 3 + 2] = s2;
                            }
                            ++cnt;
                        }
                    }
        }
        counts[i] = cnt;
        if (cnt > maxc) maxc = cnt;
    }
    return maxc > cap ? -maxc : maxc;
}

/* Uniform grid for large periodic N (SURVEY 8(d) "Oracle timing"): bins of edge >= rcut, every atom
 * tests the atoms of all DISTINCT bins within +-1 in each dimension with the same predicate as the
 * brute force.  Independent of the CUDA cell list; pinned against orc_neighbors_brute in tests.
 * Periodic boxes only (box[c] >= 2*rcut required for the minimum image to be unique). */
int orc_neighbors_grid(int n, const double *xyz, const double *box, double rcut, int fp32_pred, int cap,
                       int *counts, int *list)
{
    int nb[3];
    for (int c = 0; c < 3; ++c) {
        if (!(box[c] >= 2.0 * rcut)) return -1000000000;
        nb[c] = (int)floor(box[c] / (rcut * 1.001));
        if (nb[c] < 1) nb[c] = 1;
    }
    long nbin = (long)nb[0] * nb[1] * nb[2];
    int *bin_of = (int *)malloc(sizeof(int) * n);
    int *start = (int *)calloc(nbin + 1, sizeof(int));
    int *items = (int *)malloc(sizeof(int) * n);
    for (int i = 0; i < n; ++i) {
        int b[3];
        for (int c = 0; c < 3; ++c) {
            double w = xyz[3 * i + c] - box[c] * floor(xyz[3 * i + c] / box[c]); /* wrap into [0,L) */
            b[c] = (int)floor(w / box[c] * nb[c]);
            if (b[c] >= nb[c]) b[c] = nb[c] - 1;
            if (b[c] < 0) b[c] = 0;
        }
        bin_of[i] = (b[2] * nb[1] + b[1]) * nb[0] + b[0];
        start[bin_of[i] + 1]++;
    }
    for (long k = 0; k < nbin; ++k) start[k + 1] += start[k];
    int *fill = (int *)calloc(nbin, sizeof(int));
    for (int i = 0; i < n; ++i) items[start[bin_of[i]] + fill[bin_of[i]]++] = i;
    free(fill);

    float Lf[3], invL[3];
    for (int c = 0; c < 3; ++c) { Lf[c] = (float)box[c]; invL[c] = 1.0f / Lf[c]; }
    float rl = (float)rcut;
    float rl2 = rl * rl;
    int maxc = 0;
#pragma omp parallel for schedule(dynamic, 64) reduction(max : maxc)
    for (int i = 0; i < n; ++i) {
        int bi = bin_of[i];
        int b0 = bi % nb[0], b1 = (bi / nb[0]) % nb[1], b2 = bi / (nb[0] * nb[1]);
        int bb[3] = {b0, b1, b2};
        int cand[3][3], nc[3];
        for (int c = 0; c < 3; ++c) { /* distinct bins among b-1, b, b+1 (mod nb) */
            nc[c] = 0;
            for (int o = -1; o <= 1; ++o) {
                int v = ((bb[c] + o) % nb[c] + nb[c]) % nb[c];
                int dup = 0;
                for (int q = 0; q < nc[c]; ++q) if (cand[c][q] == v) dup = 1;
                if (!dup) cand[c][nc[c]++] = v;
            }
        }
        int cnt = 0;
        float xi[3] = {(float)xyz[3 * i], (float)xyz[3 * i + 1], (float)xyz[3 * i + 2]};
        for (int a2 = 0; a2 < nc[2]; ++a2)
            for (int a1 = 0; a1 < nc[1]; ++a1)
                for (int a0 = 0; a0 < nc[0]; ++a0) {
                    long b = ((long)cand[2][a2] * nb[1] + cand[1][a1]) * nb[0] + cand[0][a0];
                    for (int q = start[b]; q < start[b + 1]; ++q) {
                        int j = items[q];
                        if (j == i) continue;
                        int in;
                        if (fp32_pred) {
                            float xj[3] = {(float)xyz[3 * j], (float)xyz[3 * j + 1], (float)xyz[3 * j + 2]};
                            in = within_f32(xi, xj, Lf, invL, rl2);
                        } else {
                            double d[3];
                            disp(xyz + 3 * i, xyz + 3 * j, box, d);
                            in = (d[0] * d[0] + d[1] * d[1] + d[2] * d[2]) < rcut * rcut;
                        }
                        if (in) { if (cnt < cap) list[(long)i * cap + cnt] = j; ++cnt; }
                    }
                }
        counts[i] = cnt;
        if (cnt > maxc) maxc = cnt;
    }
    free(bin_of); free(start); free(items);
    return maxc > cap ? -maxc : maxc;
}

/* ---- O2/O3 pieces ------------------------------------------------------------------------ */
/* Cosine switch ("cosine function as used in ANI"), reading A4: 0 for r >= R. */
double orc_fc(double r, double R) { return r < R ? 0.5 * cos(M_PI * r / R) + 0.5 : 0.0; }
static double dfc(double r, double R) { return r < R ? -0.5 * M_PI / R * sin(M_PI * r / R) : 0.0; }

/* O4: CELU_alpha(x) = max(0,x) + min(0, alpha(exp(x/alpha)-1)) */
double orc_celu(double x, double alpha) { return x > 0.0 ? x : alpha * (exp(x / alpha) - 1.0); }
static double dcelu(double x, double alpha) { return x > 0.0 ? 1.0 : exp(x / alpha); }

/* O4: one species network forward; optionally O6 backward to the input gradient.
 * h0 = G (length widths[0]); z_l = W_l^T h_{l-1} + b_l; h_l = CELU(z_l) for l < n_layers; output = z_last. */
static double mlp_eval(const orc_model *m, int net, int s, const double *G, double *grad /* or NULL */)
{
    const int nl = m->n_layers;
    const int *w = m->widths + s * (nl + 1);
    int maxw = 0;
    for (int l = 0; l <= nl; ++l) if (w[l] > maxw) maxw = w[l];
    double *h = (double *)malloc(sizeof(double) * (size_t)(nl + 1) * maxw); /* h[l] */
    double *z = (double *)malloc(sizeof(double) * (size_t)(nl + 1) * maxw); /* z[l] */
    memcpy(h, G, sizeof(double) * w[0]);
    for (int l = 1; l <= nl; ++l) {
        const double *W = layer_ptr(m, net, s, l - 1);
        const double *b = W + (long)w[l - 1] * w[l];
        const double *hin = h + (size_t)(l - 1) * maxw;
        double *zl = z + (size_t)l * maxw, *hl = h + (size_t)l * maxw;
        for (int o = 0; o < w[l]; ++o) zl[o] = b[o];
        for (int i = 0; i < w[l - 1]; ++i) {
            double hi = hin[i];
            const double *Wi = W + (long)i * w[l];
            for (int o = 0; o < w[l]; ++o) zl[o] += Wi[o] * hi;
        }
        for (int o = 0; o < w[l]; ++o) hl[o] = (l < nl) ? orc_celu(zl[o], m->celu_alpha) : zl[o];
    }
    double out = z[(size_t)nl * maxw]; /* widths[nl] == 1 */
    if (grad) {
        /* dE/dz_last = 1; dE/dh_{l-1} = W_l dE/dz_l; dE/dz_l = dE/dh_l * CELU'(z_l) */
        double *dz = (double *)malloc(sizeof(double) * maxw);
        double *dh = (double *)malloc(sizeof(double) * maxw);
        dz[0] = 1.0;
        for (int l = nl; l >= 1; --l) {
            const double *W = layer_ptr(m, net, s, l - 1);
            for (int i = 0; i < w[l - 1]; ++i) {
                double acc = 0.0;
                for (int o = 0; o < w[l]; ++o) acc += W[(long)i * w[l] + o] * dz[o];
                dh[i] = acc;
            }
            if (l - 1 >= 1) {
                const double *zl = z + (size_t)(l - 1) * maxw;
                for (int i = 0; i < w[l - 1]; ++i) dz[i] = dh[i] * dcelu(zl[i], m->celu_alpha);
            }
        }
        for (int i = 0; i < w[0]; ++i) grad[i] = dh[i];
        free(dz); free(dh);
    }
    free(h); free(z);
    return out;
}

/* Exposed for the MLP pins (vs numpy matmul). */
double orc_mlp(const orc_model *m, int net, int species, const double *G, double *grad)
{
    return mlp_eval(m, net, species, G, grad);
}

/* O2 + O3: AEV of atom i from its radial list (ids with r < rcr); angular neighbours are the subset
 * with r < rca (PAPER.md L51-55 GraphFilter / GraphAngularExtension). */
/* displacement of list entry a (atom j) of centre i: minimum image in an orthorhombic box, or the entry's own image
 * shift shf[3 a .. 3 a + 2] in a general cell (shf != NULL) */
#define NBR_DISP(a_, j_, out_)                                                                  \
    do {                                                                                         \
        if (shf) disp_cell(xyz + 3 * i, xyz + 3 * (j_), cell, shf + 3 * (a_), out_);             \
        else disp(xyz + 3 * i, xyz + 3 * (j_), box, out_);                                       \
    } while (0)

static void aev_atom(const orc_model *m, int i, const int *species, const double *xyz, const double *box,
                     const double *cell, const int *shf, int nn, const int *nbr, double *G)
{
    const int S = m->n_species, nr = m->n_shf_r, na = m->n_shf_a, nz = m->n_shf_z;
    const int len = orc_aev_len(m), rad = S * nr;
    for (int q = 0; q < len; ++q) G[q] = 0.0;
    for (int a = 0; a < nn; ++a) {
        int j = nbr[a];
        double d[3]; NBR_DISP(a, j, d);
        double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
        if (!(r < m->rcr)) continue;
        double f = orc_fc(r, m->rcr);
        for (int k = 0; k < nr; ++k)
            G[species[j] * nr + k] += 0.25 * exp(-m->eta_r * (r - m->shf_r[k]) * (r - m->shf_r[k])) * f;
    }
    for (int a = 0; a < nn; ++a) {
        int j = nbr[a];
        double dj[3]; NBR_DISP(a, j, dj);
        double rj = sqrt(dj[0] * dj[0] + dj[1] * dj[1] + dj[2] * dj[2]);
        if (!(rj < m->rca)) continue;
        for (int b = a + 1; b < nn; ++b) { /* unordered pairs {j,k} */
            int k = nbr[b];
            double dk[3]; NBR_DISP(b, k, dk);
            double rk = sqrt(dk[0] * dk[0] + dk[1] * dk[1] + dk[2] * dk[2]);
            if (!(rk < m->rca)) continue;
            double c = (dj[0] * dk[0] + dj[1] * dk[1] + dj[2] * dk[2]) / (rj * rk);
            double th = acos(0.95 * c);
            double rb = 0.5 * (rj + rk);
            double ff = orc_fc(rj, m->rca) * orc_fc(rk, m->rca);
            int p = orc_pair_index(S, species[j], species[k]);
            for (int ia = 0; ia < na; ++ia) {
                double R = exp(-m->eta_a * (rb - m->shf_a[ia]) * (rb - m->shf_a[ia]));
                for (int iz = 0; iz < nz; ++iz) {
                    double A = pow(0.5 * (1.0 + cos(th - m->shf_z[iz])), m->zeta);
                    G[rad + (p * na + ia) * nz + iz] += 2.0 * A * R * ff;
                }
            }
        }
    }
}

/* O6: given g = dE/dG_i, add -dE/dx to F for atom i and its neighbours. */
static void aev_atom_backward(const orc_model *m, int i, const int *species, const double *xyz, const double *box,
                              const double *cell, const int *shf, int nn, const int *nbr, const double *g, double *F, double *W /* NULL or [10]: strain derivative sum d_a dE/dd_b (9) and sum |d_a dE/dd_b| */)
{
    const int S = m->n_species, nr = m->n_shf_r, na = m->n_shf_a, nz = m->n_shf_z;
    const int rad = S * nr;
    double Fi[3] = {0, 0, 0};
    for (int a = 0; a < nn; ++a) {
        int j = nbr[a];
        double d[3]; NBR_DISP(a, j, d);
        double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
        if (!(r < m->rcr)) continue;
        double f = orc_fc(r, m->rcr), fp = dfc(r, m->rcr);
        double dEdr = 0.0;
        for (int k = 0; k < nr; ++k) {
            double u = r - m->shf_r[k];
            double e = exp(-m->eta_r * u * u);
            dEdr += g[species[j] * nr + k] * 0.25 * e * (-2.0 * m->eta_r * u * f + fp);
        }
        for (int c = 0; c < 3; ++c) {
            double v = dEdr * d[c] / r; /* dE/dd_ij ; d_ij = x_j - x_i */
#pragma omp atomic
            F[3 * j + c] -= v;
            Fi[c] += v;
            if (W) for (int a2 = 0; a2 < 3; ++a2) { W[3 * a2 + c] += d[a2] * v; W[9] += fabs(d[a2] * v); }
        }
    }
    for (int a = 0; a < nn; ++a) {
        int j = nbr[a];
        double dj[3]; NBR_DISP(a, j, dj);
        double rj = sqrt(dj[0] * dj[0] + dj[1] * dj[1] + dj[2] * dj[2]);
        if (!(rj < m->rca)) continue;
        for (int b = a + 1; b < nn; ++b) {
            int k = nbr[b];
            double dk[3]; NBR_DISP(b, k, dk);
            double rk = sqrt(dk[0] * dk[0] + dk[1] * dk[1] + dk[2] * dk[2]);
            if (!(rk < m->rca)) continue;
            double c = (dj[0] * dk[0] + dj[1] * dk[1] + dj[2] * dk[2]) / (rj * rk);
            double th = acos(0.95 * c);
            double dth_dc = -0.95 / sqrt(1.0 - 0.9025 * c * c);
            double rb = 0.5 * (rj + rk);
            double fj = orc_fc(rj, m->rca), fk = orc_fc(rk, m->rca);
            double fjp = dfc(rj, m->rca), fkp = dfc(rk, m->rca);
            int p = orc_pair_index(S, species[j], species[k]);
            double dE_dth = 0.0, dE_drb = 0.0, dE_dff = 0.0; /* ff = fj*fk */
            for (int ia = 0; ia < na; ++ia) {
                double u = rb - m->shf_a[ia];
                double R = exp(-m->eta_a * u * u);
                double dR = -2.0 * m->eta_a * u * R;
                for (int iz = 0; iz < nz; ++iz) {
                    double w = g[rad + (p * na + ia) * nz + iz];
                    double base = 0.5 * (1.0 + cos(th - m->shf_z[iz]));
                    double A = pow(base, m->zeta);
                    double dA = -0.5 * m->zeta * sin(th - m->shf_z[iz]) * pow(base, m->zeta - 1.0);
                    dE_dth += w * 2.0 * dA * R * fj * fk;
                    dE_drb += w * 2.0 * A * dR * fj * fk;
                    dE_dff += w * 2.0 * A * R;
                }
            }
            double dE_dc = dE_dth * dth_dc;
            double dE_drj = 0.5 * dE_drb + dE_dff * fjp * fk;
            double dE_drk = 0.5 * dE_drb + dE_dff * fj * fkp;
            for (int q = 0; q < 3; ++q) {
                double dc_ddj = dk[q] / (rj * rk) - c * dj[q] / (rj * rj);
                double dc_ddk = dj[q] / (rj * rk) - c * dk[q] / (rk * rk);
                double vj = dE_dc * dc_ddj + dE_drj * dj[q] / rj;
                double vk = dE_dc * dc_ddk + dE_drk * dk[q] / rk;
#pragma omp atomic
                F[3 * j + q] -= vj;
#pragma omp atomic
                F[3 * k + q] -= vk;
                Fi[q] += vj + vk;
                if (W) for (int a2 = 0; a2 < 3; ++a2) {
                    W[3 * a2 + q] += dj[a2] * vj + dk[a2] * vk;
                    W[9] += fabs(dj[a2] * vj) + fabs(dk[a2] * vk);
                }
            }
        }
    }
    for (int c = 0; c < 3; ++c) {
#pragma omp atomic
        F[3 * i + c] += Fi[c];
    }
}

/* O1-O6.  nbr_method: 0 brute force, 1 grid (periodic only).  Lists are built at the exact radial
 * cutoff in fp64.  Outputs (any may be NULL except E): E[n_mols] (O5), F[n][3] (O6), e_atom[n],
 * aev[n][len], dEdG[n][len].  mol_offsets NULL => one structure.  Returns 0, or <0 on failure. */
static int energy_forces_impl(const orc_model *m, int n, const int *species, const double *xyz, const double *box,
                              const double *cell /* NULL, or 9: general cell with all images (then box is ignored) */,
                              int n_mols, const int *mol_offsets, int nbr_method, double *E, double *F,
                              double *e_atom, double *aev, double *dEdG, double *virial)
{
    const int len = orc_aev_len(m);
    const double *bx = NULL;
    if (!cell && box && (box[0] > 0.0 || box[1] > 0.0 || box[2] > 0.0)) bx = box;
    int *mol_id = (int *)malloc(sizeof(int) * (n > 0 ? n : 1));
    if (mol_offsets) {
        for (int q = 0; q < n_mols; ++q)
            for (int i = mol_offsets[q]; i < mol_offsets[q + 1]; ++i) mol_id[i] = q;
    } else {
        n_mols = 1;
        for (int i = 0; i < n; ++i) mol_id[i] = 0;
    }
    for (int q = 0; q < n_mols; ++q) E[q] = 0.0;
    if (F) memset(F, 0, sizeof(double) * 3 * (size_t)n);
    if (n == 0) { free(mol_id); return 0; }

    int cap = 64, rc;
    int *counts = (int *)malloc(sizeof(int) * n), *list = NULL, *shifts = NULL;
    for (;;) {
        list = (int *)malloc(sizeof(int) * (size_t)n * cap);
        if (cell) shifts = (int *)malloc(sizeof(int) * 3 * (size_t)n * cap);
        if (cell) rc = orc_neighbors_cell(n, xyz, cell, mol_offsets ? mol_id : NULL, m->rcr, cap, counts, list, shifts);
        else if (nbr_method == 1 && bx) rc = orc_neighbors_grid(n, xyz, bx, m->rcr, 0, cap, counts, list);
        else rc = orc_neighbors_brute(n, xyz, bx, mol_offsets ? mol_id : NULL, m->rcr, 0, cap, counts, list);
        if (rc >= 0) break;
        free(list); free(shifts); shifts = NULL;
        if (rc <= -1000000000) { free(counts); free(mol_id); return -1; }
        cap = -rc + 8;
    }
    int fail = 0;
#pragma omp parallel
    {
        double *G = (double *)malloc(sizeof(double) * len);
        double *g = (double *)malloc(sizeof(double) * len);
        double *gn = (double *)malloc(sizeof(double) * len);
        double Wt[10] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
#pragma omp for schedule(dynamic, 16)
        for (int i = 0; i < n; ++i) {
            int s = species[i];
            if (s < 0 || s >= m->n_species) { fail = 1; continue; }
            aev_atom(m, i, species, xyz, bx, cell, shifts ? shifts + 3 * (size_t)i * cap : NULL, counts[i], list + (size_t)i * cap, G);
            double e = 0.0;
            for (int q = 0; q < len; ++q) g[q] = 0.0;
            for (int net = 0; net < m->n_nets; ++net) { /* reading B5: mean over the ensemble */
                e += mlp_eval(m, net, s, G, (F || dEdG) ? gn : NULL);
                if (F || dEdG) for (int q = 0; q < len; ++q) g[q] += gn[q];
            }
            e /= m->n_nets;
            for (int q = 0; q < len; ++q) g[q] /= m->n_nets;
            if (m->self_energy) e += m->self_energy[s];
            if (e_atom) e_atom[i] = e;
            if (aev) memcpy(aev + (size_t)i * len, G, sizeof(double) * len);
            if (dEdG) memcpy(dEdG + (size_t)i * len, g, sizeof(double) * len);
#pragma omp atomic
            E[mol_id[i]] += e;
            if (F) aev_atom_backward(m, i, species, xyz, bx, cell, shifts ? shifts + 3 * (size_t)i * cap : NULL, counts[i], list + (size_t)i * cap, g, F, virial ? Wt : NULL);
        }
        if (virial)
            for (int q = 0; q < 10; ++q) {
#pragma omp atomic
                virial[q] += Wt[q];
            }
        free(G); free(g); free(gn);
    }
    free(counts); free(list); free(shifts); free(mol_id);
    return fail ? -2 : 0;
}

int orc_energy_forces(const orc_model *m, int n, const int *species, const double *xyz, const double *box,
                      int n_mols, const int *mol_offsets, int nbr_method, double *E, double *F,
                      double *e_atom, double *aev, double *dEdG)
{
    return energy_forces_impl(m, n, species, xyz, box, NULL, n_mols, mol_offsets, nbr_method, E, F, e_atom, aev, dEdG, NULL);
}

/* The same in a general cell (rows a, b, c) with all periodic images; virial [10] as orc_energy_forces_virial or NULL
 * (one structure). */
int orc_energy_forces_cell(const orc_model *m, int n, const int *species, const double *xyz, const double *cell,
                           int n_mols, const int *mol_offsets, double *E, double *F, double *e_atom, double *aev,
                           double *virial)
{
    if (virial) for (int q = 0; q < 10; ++q) virial[q] = 0.0;
    return energy_forces_impl(m, n, species, xyz, NULL, cell, n_mols, mol_offsets, 0, E, F, e_atom, aev, NULL, virial);
}

/* NEXT-2 (first part; "energy_and_forces_and_virial"): the energy depends on
 * the coordinates (and, under PBC, the cell) only through the displacement vectors d it is built from -- d_ij of every
 * radial term and d_ij, d_ik of every angular term -- so under a homogeneous deformation x -> (1 + eps) x,
 * cell -> (1 + eps) cell every d -> (1 + eps) d and
 *     V_ab = dE/d eps_ab = sum over those d of d_a (dE/dd)_b          (the virial; stress = V / volume).
 * One structure only.  virial[0..8] = V (row-major, symmetric up to rounding because E is rotation invariant),
 * virial[9] = sum |d_a (dE/dd)_b|, the scale against which rounding errors of an fp32 evaluation are judged. */
int orc_energy_forces_virial(const orc_model *m, int n, const int *species, const double *xyz, const double *box,
                             int nbr_method, double *E, double *F, double *virial /*[10]*/)
{
    for (int q = 0; q < 10; ++q) virial[q] = 0.0;
    return energy_forces_impl(m, n, species, xyz, box, NULL, 1, NULL, nbr_method, E, F, NULL, NULL, NULL, virial);
}

/* O7 rebuild rule (reading C2): max_i |x_i - xref_i| > skin/2 (strict). */
int orc_needs_rebuild(int n, const double *xyz, const double *xref, double skin)
{
    double lim2 = 0.25 * skin * skin;
    for (int i = 0; i < n; ++i) {
        double d0 = xyz[3 * i] - xref[3 * i], d1 = xyz[3 * i + 1] - xref[3 * i + 1], d2 = xyz[3 * i + 2] - xref[3 * i + 2];
        if (d0 * d0 + d1 * d1 + d2 * d2 > lim2) return 1;
    }
    return 0;
}

/* O7: velocity Verlet (NVE "reverts to the velocity Verlet integrator").
 * a = accel_conv * F / m.  Per step: v += dt/2 a; x += dt v; [rebuild test]; F(x); v += dt/2 a.
 * Coordinates are not wrapped.  Forces are evaluated with exact (fresh) lists every step -- in exact
 * arithmetic a valid skinned list gives the same E,F -- but the rebuild rule is tracked so that
 * n_rebuilds reports what an implementation using a Verlet skin must do (the initial build counts as 1).
 * F_io: forces at the input positions if have_forces, else computed here; holds the final forces on return.
 * epot/ekin: [n_steps+1] values at steps 0..n_steps (may be NULL). */
static int md_impl(const orc_model *m, int n, const int *species, double *xyz, double *vel, double *F_io, int have_forces,
                   const double *mass /*[S]*/, const double *box, const double *cell, double dt, double accel_conv, int n_steps,
                   double skin, int nbr_method, double *epot, double *ekin, int *n_rebuilds)
{
    double E;
    int rc = 0, nreb = 1;
    double *xref = (double *)malloc(sizeof(double) * 3 * (size_t)n);
    memcpy(xref, xyz, sizeof(double) * 3 * (size_t)n);
    if (!have_forces || epot) {
        rc = energy_forces_impl(m, n, species, xyz, box, cell, 1, NULL, nbr_method, &E, F_io, NULL, NULL, NULL, NULL);
        if (rc) { free(xref); return rc; }
    }
    for (int step = 0;; ++step) {
        if (ekin) {
            double k = 0.0;
            for (int i = 0; i < n; ++i)
                k += 0.5 * mass[species[i]] * (vel[3 * i] * vel[3 * i] + vel[3 * i + 1] * vel[3 * i + 1] + vel[3 * i + 2] * vel[3 * i + 2]);
            ekin[step] = k / accel_conv;
        }
        if (epot) epot[step] = E;
        if (step == n_steps) break;
        for (int i = 0; i < n; ++i)
            for (int c = 0; c < 3; ++c) {
                vel[3 * i + c] += 0.5 * dt * accel_conv * F_io[3 * i + c] / mass[species[i]];
                xyz[3 * i + c] += dt * vel[3 * i + c];
            }
        if (orc_needs_rebuild(n, xyz, xref, skin)) { memcpy(xref, xyz, sizeof(double) * 3 * (size_t)n); ++nreb; }
        rc = energy_forces_impl(m, n, species, xyz, box, cell, 1, NULL, nbr_method, &E, F_io, NULL, NULL, NULL, NULL);
        if (rc) break;
        for (int i = 0; i < n; ++i)
            for (int c = 0; c < 3; ++c) vel[3 * i + c] += 0.5 * dt * accel_conv * F_io[3 * i + c] / mass[species[i]];
    }
    if (n_rebuilds) *n_rebuilds = nreb;
    free(xref);
    return rc;
}

int orc_md(const orc_model *m, int n, const int *species, double *xyz, double *vel, double *F_io, int have_forces,
           const double *mass /*[S]*/, const double *box, double dt, double accel_conv, int n_steps, double skin,
           int nbr_method, double *epot, double *ekin, int *n_rebuilds)
{
    return md_impl(m, n, species, xyz, vel, F_io, have_forces, mass, box, NULL, dt, accel_conv, n_steps, skin, nbr_method, epot, ekin,
                   n_rebuilds);
}

/* O7 in a general cell with all images (orc_energy_forces_cell). */
int orc_md_cell(const orc_model *m, int n, const int *species, double *xyz, double *vel, double *F_io, int have_forces,
                const double *mass /*[S]*/, const double *cell, double dt, double accel_conv, int n_steps, double skin,
                double *epot, double *ekin, int *n_rebuilds)
{
    return md_impl(m, n, species, xyz, vel, F_io, have_forces, mass, NULL, cell, dt, accel_conv, n_steps, skin, 0, epot, ekin, n_rebuilds);
}

/* ---- NEXT-1: Langevin dynamics, BAOAB splitting.  PAPER.md L307: the MD engine offers
 * "Langevin dynamics (using the BAOAB scheme)"; L323: every benchmark of the paper runs "Langevin 300 K".
 * Per step (Leimkuhler & Matthews 2013, the scheme the paper names):
 *   B: v += dt/2 a(F)      A: x += dt/2 v      O: v = c1 v + c2_s xi,  c1 = exp(-gamma dt),
 *   A: x += dt/2 v         [rebuild test]      F(x)     B: v += dt/2 a(F)      c2_s = sqrt((1 - c1^2) kT accel_conv / m_s)
 * xi: three independent standard normals per atom and step from a counter-based generator, so that the CUDA path can
 * draw the same numbers: Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11) with counter (atom index, step, 0, 0) and
 * key (seed low, seed high); uniforms u = ((r >> 9) + 1/2) 2^-23 (exact in fp32 and fp64), Box-Muller
 * xi_0 = sqrt(-2 ln u_0) cos(2 pi u_1), xi_1 = sqrt(-2 ln u_0) sin(2 pi u_1), xi_2 = sqrt(-2 ln u_2) cos(2 pi u_3).
 * gamma = 0 gives c1 = 1, c2 = 0: velocity Verlet (pinned against orc_md). */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        if (round) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

void orc_langevin_normals(uint32_t atom, uint32_t step, uint64_t seed, double xi[3])
{
    const uint32_t ctr[4] = {atom, step, 0u, 0u}, key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    uint32_t r[4];
    double u[4];
    orc_philox4x32_10(ctr, key, r);
    for (int q = 0; q < 4; ++q) u[q] = ((double)(r[q] >> 9) + 0.5) / 8388608.0;
    const double a = sqrt(-2.0 * log(u[0])), b = sqrt(-2.0 * log(u[2]));
    xi[0] = a * cos(2.0 * M_PI * u[1]);
    xi[1] = a * sin(2.0 * M_PI * u[1]);
    xi[2] = b * cos(2.0 * M_PI * u[3]);
}

/* Same arguments as orc_md plus gamma [1/time], kT [energy], seed, step0 (counter of the first step). */
int orc_md_langevin(const orc_model *m, int n, const int *species, double *xyz, double *vel, double *F_io, int have_forces,
                    const double *mass /*[S]*/, const double *box, double dt, double accel_conv, int n_steps, double skin,
                    int nbr_method, double gamma, double kT, uint64_t seed, uint32_t step0, double *epot, double *ekin,
                    int *n_rebuilds)
{
    double E;
    int rc = 0, nreb = 1;
    const double c1 = exp(-gamma * dt);
    double *xref = (double *)malloc(sizeof(double) * 3 * (size_t)n);
    memcpy(xref, xyz, sizeof(double) * 3 * (size_t)n);
    if (!have_forces || epot) {
        rc = orc_energy_forces(m, n, species, xyz, box, 1, NULL, nbr_method, &E, F_io, NULL, NULL, NULL);
        if (rc) { free(xref); return rc; }
    }
    for (int step = 0;; ++step) {
        if (ekin) {
            double k = 0.0;
            for (int i = 0; i < n; ++i)
                k += 0.5 * mass[species[i]] * (vel[3 * i] * vel[3 * i] + vel[3 * i + 1] * vel[3 * i + 1] + vel[3 * i + 2] * vel[3 * i + 2]);
            ekin[step] = k / accel_conv;
        }
        if (epot) epot[step] = E;
        if (step == n_steps) break;
        for (int i = 0; i < n; ++i) {
            const double ms = mass[species[i]];
            const double c2 = sqrt((1.0 - c1 * c1) * kT * accel_conv / ms);
            double xi[3];
            orc_langevin_normals((uint32_t)i, step0 + (uint32_t)step, seed, xi);
            for (int c = 0; c < 3; ++c) {
                vel[3 * i + c] += 0.5 * dt * accel_conv * F_io[3 * i + c] / ms; /* B */
                xyz[3 * i + c] += 0.5 * dt * vel[3 * i + c];                    /* A */
                vel[3 * i + c] = c1 * vel[3 * i + c] + c2 * xi[c];              /* O */
                xyz[3 * i + c] += 0.5 * dt * vel[3 * i + c];                    /* A */
            }
        }
        if (orc_needs_rebuild(n, xyz, xref, skin)) { memcpy(xref, xyz, sizeof(double) * 3 * (size_t)n); ++nreb; }
        rc = orc_energy_forces(m, n, species, xyz, box, 1, NULL, nbr_method, &E, F_io, NULL, NULL, NULL);
        if (rc) break;
        for (int i = 0; i < n; ++i)
            for (int c = 0; c < 3; ++c) vel[3 * i + c] += 0.5 * dt * accel_conv * F_io[3 * i + c] / mass[species[i]]; /* B */
    }
    if (n_rebuilds) *n_rebuilds = nreb;
    free(xref);
    return rc;
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
