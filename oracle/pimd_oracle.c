/*
 * pimd_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of one ring-polymer PIMD step over all P beads
 * (neighbour list -> GFN-style direct-force network -> normal-mode propagation
 * + PILE-L), written from /root/reference/PAPER.md ("P:Lnnn") and the readings
 * fixed in SURVEY.md section 8(c) / DESIGN.md.  It shares no code with the CUDA path
 * under paper_2503_23728_b200/ and must only be imported / linked / executed by
 * tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference.
 *
 * Everything is written in the paper's order and notation, without blocking,
 * fusion or algebraic shortcuts:
 *   - neighbour list: brute-force O(N^2) definition AND a cell list (L1-L4); tests
 *     assert the two are identical.
 *   - GFN: the LITERAL recursion of P:L74 with a stored per-pair edge state
 *     e_ij^(l) (the CUDA path uses an algebraically equivalent running-sum form;
 *     parity between the two is therefore also a check of that algebra).
 *   - integrator: O(dt/2) B(dt/2) A(dt) [forces] B(dt/2) O(dt/2) (N3) with the
 *     normal-mode matrix of N2 and Philox4x32-10 + Box-Muller noise (N4).
 *
 * Parity pins (tests/test_oracle_*.py): Philox known answers; C.C^T = I and
 * C^T K C diagonal; exact free-ring-polymer energy conservation; NVE bounded
 * fluctuation; P=1 == velocity Verlet; finite-P harmonic-oscillator energy
 * (P:L358 corrected, -> P:L350); cell list == brute force; ice-Ic shell counts;
 * sum F = 0, sum r x F = 0, rotation/translation/permutation equivariance,
 * image-shift invariance, L=0 two-atom hand evaluation, independent dense numpy
 * evaluation.  The network's numerical OUTPUT has no value printed in the paper:
 * "parity unpinned by the paper" -- pinned by the invariants above only.
 *
 * Build: gcc -O3 -ffp-contract=off -fopenmp -shared -fPIC (see oracle/build.py).
 * -ffp-contract=off keeps the neighbour predicate free of fused multiply-adds (L3).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* CODATA 2018 */
#define KB_EV 8.617333262145e-5   /* eV / K */
#define HBAR_EVFS 0.658211956548  /* eV fs */
#define AMU_INTERNAL 103.6426965268 /* 1 amu A^2/fs^2 in eV */

typedef struct {
    int32_t kind;      /* 0 GFN, 1 harmonic well, 2 free ring polymer */
    int32_t n_species, n_rbf, hidden, n_layers;
    double r_cut, agg_norm, force_scale, harmonic_omega;
    const float *weights;
    int64_t n_weights;
} ref_net_params;

typedef struct {
    double k_prim, k_vir, k_cvir, v_pot, t_centroid;
} ref_estimators_t;

typedef struct {
    int N, R, P, periodic;
    double box[3];
    int32_t *species;
    double *mass; /* [N], internal units eV fs^2 / A^2 */
    double T, dt, gamma_fs;
    uint64_t seed;
    int64_t step;
    ref_net_params net;
    /* weights promoted to fp64, stored transposed [in][out] (layout only; every
       sum over the input index still runs in ascending order) */
    double *Emb, *We1, *be1, *We2, *be2;
    double **Ws, **Wvn, **Wvm, **bv1, **Wv2, **bv2, **Wa, **ba;
    double *Wf1, *bf1, *wf2, bf2;
    double *q, *p, *F; /* [R][P][N][3] */
    double *Fgross;    /* [R][P][N] diagnostic: sum of the magnitudes of the terms of F_i */
    double *C;         /* [P][P], C[j*P+k], bead j, mode k */
    double *omega_k;   /* [P] */
    int forces_valid;
    /* well-tempered metadynamics: one bias V_G(s) per replica, felt by every bead */
    int md_cv;                   /* 0 off, 1 s_dimer, 2 Debye XRD intensity */
    int md_atoms[6];             /* s_dimer: O1, H1, O2, O4, H2, O3 */
    double md_f[16], md_Q;       /* Debye: scattering factor per species, Q = 4 pi sin(theta) / lambda */
    double md_sigma, md_w0, md_biasf;
    int md_every, md_max, *md_n; /* deposition stride (steps), capacity, Gaussians deposited per replica [R] */
    double *md_c, *md_h;         /* [R][md_max] centres and heights */
    double *md_s, *md_ds;        /* [R][P] CV of every bead; [R][P][N][3] its gradient */
    int transform;  /* 0 normal modes (N2), 1 staging, 2 primitive (no transformation, explicit spring forces) */
    int thermostat; /* 0 PILE-L / white-noise Langevin, 1 PILE-G (global velocity rescaling of the free mode) */
} ref_ctx;

/* ------------------------------------------------------------------ */
/* Philox4x32-10 (N4)                                                   */
/* ------------------------------------------------------------------ */
void ref_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        if (r > 0) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* three standard normals for (atom, r*P+mode, step, tag): Box-Muller in fp64 (N4) */
void ref_normal3(uint64_t seed, uint32_t atom, uint32_t sysmode, uint32_t step, uint32_t tag, double xi[3])
{
    uint32_t ctr[4] = {atom, sysmode, step, tag};
    uint32_t key[2] = {(uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32)};
    uint32_t x[4];
    ref_philox4x32_10(ctr, key, x);
    const double s = 1.0 / 4294967296.0;
    double ua = ((double)x[0] + 0.5) * s, ub = ((double)x[1] + 0.5) * s;
    double uc = ((double)x[2] + 0.5) * s, ud = ((double)x[3] + 0.5) * s;
    double ra = sqrt(-2.0 * log(ua)), rc = sqrt(-2.0 * log(uc));
    const double two_pi = 6.283185307179586476925286766559;
    xi[0] = ra * cos(two_pi * ub);
    xi[1] = ra * sin(two_pi * ub);
    xi[2] = rc * cos(two_pi * ud);
}

/* ------------------------------------------------------------------ */
/* normal-mode matrix (N2)                                              */
/* ------------------------------------------------------------------ */
void ref_nm_matrix(int P, double *C)
{
    const double pi = 3.14159265358979323846264338327950288;
    for (int j = 0; j < P; ++j)
        for (int k = 0; k < P; ++k) {
            double v;
            if (k == 0) v = 1.0 / sqrt((double)P);
            else if (2 * k < P) v = sqrt(2.0 / P) * cos(2.0 * pi * j * k / P);
            else if (2 * k == P) v = ((j % 2) ? -1.0 : 1.0) / sqrt((double)P);
            else v = sqrt(2.0 / P) * sin(2.0 * pi * j * k / P);
            C[j * P + k] = v;
        }
}

/* ------------------------------------------------------------------ */
/* neighbour lists (L1-L4)                                              */
/* ------------------------------------------------------------------ */
/* L3 predicate: fixed operation order, no contraction.  Returns d2, writes delta = q_j - q_i (min image). */
static double min_image_d2(const double *qi, const double *qj, const double box[3], int periodic, double d[3])
{
    for (int a = 0; a < 3; ++a) {
        double dx = qj[a] - qi[a];
        if (periodic) dx = dx - box[a] * round(dx / box[a]);
        d[a] = dx;
    }
    return (d[0] * d[0] + d[1] * d[1]) + d[2] * d[2];
}

/* brute force, one bead-system.  row_ptr[N+1]; col capacity cap.  Returns pair count or -1 on overflow. */
int64_t ref_nlist_brute(int N, const double *q, const double box[3], double r_cut, int32_t *row_ptr, int32_t *col,
                        int64_t cap)
{
    int periodic = box[0] > 0.0;
    double rc2 = r_cut * r_cut, d[3];
    int64_t n = 0;
    for (int i = 0; i < N; ++i) {
        row_ptr[i] = (int32_t)n;
        for (int j = 0; j < N; ++j) {
            if (j == i) continue;
            if (min_image_d2(q + 3 * i, q + 3 * j, box, periodic, d) < rc2) {
                if (n >= cap) return -1;
                col[n++] = j;
            }
        }
    }
    row_ptr[N] = (int32_t)n;
    return n;
}

static int cmp_i32(const void *a, const void *b)
{
    int32_t x = *(const int32_t *)a, y = *(const int32_t *)b;
    return (x > y) - (x < y);
}

/* cell list, one bead-system (L2, L4): bin on the wrapped fraction, scan the de-duplicated stencil. */
int64_t ref_nlist_cell(int N, const double *q, const double box[3], double r_cut, int32_t *row_ptr, int32_t *col,
                       int64_t cap)
{
    int periodic = box[0] > 0.0;
    double rc2 = r_cut * r_cut, d[3];
    int nc[3] = {1, 1, 1};
    if (periodic)
        for (int a = 0; a < 3; ++a) {
            nc[a] = (int)floor(box[a] / r_cut);
            if (nc[a] < 1) nc[a] = 1;
        }
    int ncell = nc[0] * nc[1] * nc[2];
    int *cell_of = (int *)malloc(sizeof(int) * N);
    int *start = (int *)calloc(ncell + 1, sizeof(int));
    int *perm = (int *)malloc(sizeof(int) * (N > 0 ? N : 1));
    int *cxyz = (int *)malloc(sizeof(int) * 3 * (N > 0 ? N : 1));
    for (int i = 0; i < N; ++i) {
        int c[3] = {0, 0, 0};
        if (periodic)
            for (int a = 0; a < 3; ++a) {
                double x = q[3 * i + a] / box[a];
                double f = x - floor(x);
                int ci = (int)(f * nc[a]);
                if (ci > nc[a] - 1) ci = nc[a] - 1;
                c[a] = ci;
            }
        cxyz[3 * i] = c[0]; cxyz[3 * i + 1] = c[1]; cxyz[3 * i + 2] = c[2];
        cell_of[i] = (c[0] * nc[1] + c[1]) * nc[2] + c[2];
        start[cell_of[i] + 1]++;
    }
    for (int c = 0; c < ncell; ++c) start[c + 1] += start[c];
    int *cursor = (int *)malloc(sizeof(int) * (ncell > 0 ? ncell : 1));
    memcpy(cursor, start, sizeof(int) * ncell);
    for (int i = 0; i < N; ++i) perm[cursor[cell_of[i]]++] = i;

    int64_t n = 0;
    int overflow = 0;
    for (int i = 0; i < N && !overflow; ++i) {
        row_ptr[i] = (int32_t)n;
        int64_t row_begin = n;
        /* distinct neighbour cells per dimension */
        int lst[3][3] = {{0}}, cnt[3];
        for (int a = 0; a < 3; ++a) {
            cnt[a] = 0;
            for (int o = -1; o <= 1; ++o) {
                int c = cxyz[3 * i + a] + o;
                if (periodic) c = ((c % nc[a]) + nc[a]) % nc[a];
                else if (c < 0 || c >= nc[a]) continue;
                int dup = 0;
                for (int t = 0; t < cnt[a]; ++t) dup |= (lst[a][t] == c);
                if (!dup) lst[a][cnt[a]++] = c;
            }
        }
        for (int ix = 0; ix < cnt[0]; ++ix)
            for (int iy = 0; iy < cnt[1]; ++iy)
                for (int iz = 0; iz < cnt[2]; ++iz) {
                    int c = (lst[0][ix] * nc[1] + lst[1][iy]) * nc[2] + lst[2][iz];
                    for (int s = start[c]; s < start[c + 1]; ++s) {
                        int j = perm[s];
                        if (j == i) continue;
                        if (min_image_d2(q + 3 * i, q + 3 * j, box, periodic, d) < rc2) {
                            if (n >= cap) { overflow = 1; break; }
                            col[n++] = j;
                        }
                    }
                }
        qsort(col + row_begin, (size_t)(n - row_begin), sizeof(int32_t), cmp_i32);
    }
    row_ptr[N] = (int32_t)n;
    free(cell_of); free(start); free(perm); free(cxyz); free(cursor);
    return overflow ? -1 : n;
}

/* ------------------------------------------------------------------ */
/* GFN-style direct-force network (G0-G5), literal edge recursion       */
/* ------------------------------------------------------------------ */
static double silu(double x) { return x / (1.0 + exp(-x)); }

/* y[o] = sum_k Wt[k][o] * x[k] + b[o]; the sum over k runs in ascending k for every o */
static void affine(const double *Wt, const double *b, const double *x, int n_in, int n_out, double *y)
{
    for (int o = 0; o < n_out; ++o) y[o] = 0.0;
    for (int k = 0; k < n_in; ++k) {
        const double *w = Wt + (size_t)k * n_out;
        double xk = x[k];
        for (int o = 0; o < n_out; ++o) y[o] += w[o] * xk;
    }
    if (b)
        for (int o = 0; o < n_out; ++o) y[o] += b[o];
}

static int g_inner_parallel = 0;

/* forces on one bead-system from its pair list; F[N][3] in eV/A */
/* gross (may be NULL): per atom, force_scale * sum_j c_ij (sum_o |w_f2[o] SiLU(t_o)| + |b_f2|): the sum of the magnitudes
 * of every term that is added up into F_i (readout channels, then neighbours).  A diagnostic only -- the scale a
 * forward error bound of those sums is stated against; F does not depend on it. */
static void gfn_forces_system(const ref_ctx *c, const double *q, const int32_t *row_ptr, const int32_t *col, double *F,
                              double *gross)
{
    const int N = c->N, H = c->net.hidden, K = c->net.n_rbf, L = c->net.n_layers;
    const double rc = c->net.r_cut;
    const int64_t npairs = row_ptr[N];
    const double pi = 3.14159265358979323846264338327950288;
    double *n = (double *)malloc(sizeof(double) * (size_t)N * H);
    double *x = (double *)malloc(sizeof(double) * (size_t)N * H);
    double *m = (double *)malloc(sizeof(double) * (size_t)N * H);
    double *a = (double *)malloc(sizeof(double) * (size_t)N * H);
    double *e = (double *)malloc(sizeof(double) * (size_t)(npairs > 0 ? npairs : 1) * H);
    double *cw = (double *)malloc(sizeof(double) * (size_t)(npairs > 0 ? npairs : 1));
    double *uv = (double *)malloc(sizeof(double) * 3 * (size_t)(npairs > 0 ? npairs : 1));
    int32_t *pi_row = (int32_t *)malloc(sizeof(int32_t) * (size_t)(npairs > 0 ? npairs : 1));

    for (int i = 0; i < N; ++i) {
        memcpy(n + (size_t)i * H, c->Emb + (size_t)c->species[i] * H, sizeof(double) * H); /* n^0 = Emb[species] */
        for (int p = row_ptr[i]; p < row_ptr[i + 1]; ++p) pi_row[p] = i;
    }

    /* G1 + G2: geometry, RBF, cutoff, initial edge e^0_ij = W_e2 SiLU(W_e1 g + b_e1) + b_e2 */
    const double delta = rc / (K - 1);
#pragma omp parallel for schedule(static) if (g_inner_parallel)
    for (int64_t p = 0; p < npairs; ++p) {
        int i = pi_row[p], j = col[p];
        double d[3];
        double d2 = min_image_d2(q + 3 * i, q + 3 * j, c->box, c->periodic, d);
        double dist = sqrt(d2);
        double dd = dist > 1e-12 ? dist : 1e-12;
        uv[3 * p] = -d[0] / dd; uv[3 * p + 1] = -d[1] / dd; uv[3 * p + 2] = -d[2] / dd; /* (r_i - r_j)/d */
        cw[p] = 0.5 * (cos(pi * dist / rc) + 1.0);
        double g[512], h1[512];
        for (int k = 0; k < K; ++k) {
            double t = dist - k * delta;
            g[k] = exp(-(t * t) / (2.0 * delta * delta));
        }
        affine(c->We1, c->be1, g, K, H, h1);
        for (int o = 0; o < H; ++o) h1[o] = silu(h1[o]);
        affine(c->We2, c->be2, h1, H, H, e + (size_t)p * H);
    }

    /* G3: L interaction layers */
    for (int l = 0; l < L; ++l) {
#pragma omp parallel for schedule(static) if (g_inner_parallel)
        for (int j = 0; j < N; ++j) affine(c->Ws[l], NULL, n + (size_t)j * H, H, H, x + (size_t)j * H);
#pragma omp parallel for schedule(static) if (g_inner_parallel)
        for (int i = 0; i < N; ++i) {
            double *mi = m + (size_t)i * H;
            for (int o = 0; o < H; ++o) mi[o] = 0.0;
            for (int p = row_ptr[i]; p < row_ptr[i + 1]; ++p) { /* m_i = phi_m(e_ij): cutoff-weighted sum over j */
                const double *ep = e + (size_t)p * H, *xj = x + (size_t)col[p] * H;
                for (int o = 0; o < H; ++o) mi[o] += cw[p] * (ep[o] * xj[o]);
            }
            for (int o = 0; o < H; ++o) mi[o] *= c->net.agg_norm;
        }
#pragma omp parallel for schedule(static) if (g_inner_parallel)
        for (int i = 0; i < N; ++i) { /* n_i += phi_v(n_i, m_i) */
            double u[512], v[512], w[512];
            double *ni = n + (size_t)i * H;
            affine(c->Wvn[l], c->bv1[l], ni, H, H, u);
            affine(c->Wvm[l], NULL, m + (size_t)i * H, H, H, v);
            for (int o = 0; o < H; ++o) u[o] = silu(u[o] + v[o]);
            affine(c->Wv2[l], c->bv2[l], u, H, H, w);
            for (int o = 0; o < H; ++o) ni[o] += w[o];
            affine(c->Wa[l], c->ba[l], ni, H, H, a + (size_t)i * H); /* node -> edge MLP on the UPDATED node */
        }
#pragma omp parallel for schedule(static) if (g_inner_parallel)
        for (int64_t p = 0; p < npairs; ++p) { /* e_ij += agg(n_i, n_j) = a_i + a_j */
            double *ep = e + (size_t)p * H;
            const double *ai = a + (size_t)pi_row[p] * H, *aj = a + (size_t)col[p] * H;
            for (int o = 0; o < H; ++o) ep[o] += ai[o] + aj[o];
        }
    }

    /* G4: F_ij = c_ij * d_ij * phi_f(e_ij), F_i = force_scale * sum_j F_ij */
#pragma omp parallel for schedule(static) if (g_inner_parallel)
    for (int i = 0; i < N; ++i) {
        double f[3] = {0.0, 0.0, 0.0}, t[512], fg = 0.0;
        for (int p = row_ptr[i]; p < row_ptr[i + 1]; ++p) {
            affine(c->Wf1, c->bf1, e + (size_t)p * H, H, H, t);
            double s = 0.0, sa = 0.0;
            for (int o = 0; o < H; ++o) {
                double term = c->wf2[o] * silu(t[o]);
                s += term;
                sa += fabs(term);
            }
            s += c->bf2;
            for (int ax = 0; ax < 3; ++ax) f[ax] += cw[p] * s * uv[3 * p + ax];
            fg += cw[p] * (sa + fabs(c->bf2));
        }
        for (int ax = 0; ax < 3; ++ax) F[3 * i + ax] = c->net.force_scale * f[ax];
        if (gross) gross[i] = fabs(c->net.force_scale) * fg;
    }
    free(n); free(x); free(m); free(a); free(e); free(cw); free(uv); free(pi_row);
}

/* pair capacity used internally for one bead-system */
static int64_t sys_pair_cap(const ref_ctx *c) { return (int64_t)c->N * (c->N - 1) + 1; }

/* ------------------------------------------------------------------ */
/* well-tempered metadynamics with the paper's two collective variables                            */
/* ------------------------------------------------------------------ */
/* P:L164  s_dimer = d(O1,H1) - d(O2,H1) + d(O4,H2) - d(O3,H2): distances of one bead-system (no periodic image: the dimer is an
 * open cluster; with a box the minimum image is used).  grad adds +-(r_X - r_Y)/d to the six atoms. */
static double md_dist(const ref_ctx *c, const double *qs, int x, int y, double u[3])
{
    double d2 = 0.0;
    for (int a = 0; a < 3; ++a) {
        double dx = qs[(size_t)x * 3 + a] - qs[(size_t)y * 3 + a];
        if (c->periodic) dx = dx - c->box[a] * round(dx / c->box[a]);
        u[a] = dx; d2 += dx * dx;
    }
    double d = sqrt(d2);
    for (int a = 0; a < 3; ++a) u[a] /= d;
    return d;
}
static double cv_dimer(const ref_ctx *c, const double *qs, double *grad)
{
    const int *t = c->md_atoms; /* O1, H1, O2, O4, H2, O3 */
    const int pr[4][2] = {{t[0], t[1]}, {t[2], t[1]}, {t[3], t[4]}, {t[5], t[4]}};
    const double sg[4] = {1.0, -1.0, 1.0, -1.0};
    double s = 0.0;
    memset(grad, 0, sizeof(double) * (size_t)c->N * 3);
    for (int k = 0; k < 4; ++k) {
        double u[3];
        s += sg[k] * md_dist(c, qs, pr[k][0], pr[k][1], u);
        for (int a = 0; a < 3; ++a) {
            grad[(size_t)pr[k][0] * 3 + a] += sg[k] * u[a];
            grad[(size_t)pr[k][1] * 3 + a] -= sg[k] * u[a];
        }
    }
    return s;
}
/* P:L215, P:L450  s_water = (1/N) sum_i sum_j f_i f_j sin(Q R_ij) / (Q R_ij), the double sum over ALL ordered pairs including
 * i = j (sinc(0) = 1), R_ij the minimum-image distance.  d/dr_i: the ordered pairs (i,j) and (j,i) both contain r_i. */
static double cv_debye(const ref_ctx *c, const double *qs, double *grad)
{
    const int N = c->N;
    double s = 0.0;
    memset(grad, 0, sizeof(double) * (size_t)N * 3);
    for (int i = 0; i < N; ++i) {
        const double fi = c->md_f[c->species[i]];
        for (int j = 0; j < N; ++j) {
            const double fj = c->md_f[c->species[j]];
            if (j == i) { s += fi * fj; continue; }
            double u[3];
            const double R = md_dist(c, qs, i, j, u), x = c->md_Q * R;
            const double g = sin(x) / x;
            s += fi * fj * g;
            const double dg = (cos(x) - g) / R; /* d sinc(Q R) / dR */
            for (int a = 0; a < 3; ++a) grad[(size_t)i * 3 + a] += 2.0 * fi * fj * dg * u[a] / (double)N;
        }
    }
    return s / (double)N;
}
/* V_G(s) = sum_g h_g exp(-(s - c_g)^2 / (2 sigma^2))  (P:L140 with 2 sigma read as 2 sigma^2) and dV/ds */
static double md_bias(const ref_ctx *c, int r, double s, double *dVds)
{
    double V = 0.0, dV = 0.0;
    const double is2 = 1.0 / (c->md_sigma * c->md_sigma);
    for (int g = 0; g < c->md_n[r]; ++g) {
        const double d = s - c->md_c[(size_t)r * c->md_max + g];
        const double e = c->md_h[(size_t)r * c->md_max + g] * exp(-0.5 * d * d * is2);
        V += e; dV -= e * d * is2;
    }
    if (dVds) *dVds = dV;
    return V;
}
/* the bias is a potential term like any other: every bead k feels F = -dV_G/ds(s_k) grad s(q_k) */
static void metad_add_bias_forces(ref_ctx *c)
{
    const int N = c->N;
    for (int r = 0; r < c->R; ++r)
        for (int k = 0; k < c->P; ++k) {
            const size_t sys = (size_t)r * c->P + k;
            const double *qs = c->q + sys * N * 3;
            double *gr = c->md_ds + sys * N * 3;
            const double s = (c->md_cv == 1) ? cv_dimer(c, qs, gr) : cv_debye(c, qs, gr);
            c->md_s[sys] = s;
            double dV;
            md_bias(c, r, s, &dV);
            for (size_t t = 0; t < (size_t)N * 3; ++t) c->F[sys * N * 3 + t] -= dV * gr[t];
        }
}
/* deposition: every md_every steps one Gaussian per bead at the bead's CV value, height
 * (w0 / P) exp(-beta V_G(s_k) / (gamma - 1)) with V_G the bias BEFORE this deposition event and beta = 1 / k_B T */
static void metad_deposit(ref_ctx *c)
{
    const double kT = KB_EV * c->T;
    for (int r = 0; r < c->R; ++r) {
        const int n0 = c->md_n[r];
        double hs[1024];
        for (int k = 0; k < c->P; ++k)
            hs[k] = (c->md_w0 / c->P) * exp(-md_bias(c, r, c->md_s[(size_t)r * c->P + k], NULL) / (kT * (c->md_biasf - 1.0)));
        for (int k = 0; k < c->P && n0 + k < c->md_max; ++k) {
            c->md_c[(size_t)r * c->md_max + n0 + k] = c->md_s[(size_t)r * c->P + k];
            c->md_h[(size_t)r * c->md_max + n0 + k] = hs[k];
        }
        c->md_n[r] = (n0 + c->P <= c->md_max) ? n0 + c->P : c->md_max;
    }
}

static int compute_forces(ref_ctx *c)
{
    const int N = c->N, nsys = c->R * c->P;
    int overflow = 0;
    if (c->net.kind == 2) {
        memset(c->F, 0, sizeof(double) * (size_t)nsys * N * 3);
    } else if (c->net.kind == 1) { /* V = 1/2 m w^2 |r|^2 per atom */
        double w2 = c->net.harmonic_omega * c->net.harmonic_omega;
        for (int s = 0; s < nsys; ++s)
            for (int i = 0; i < N; ++i)
                for (int a = 0; a < 3; ++a) {
                    size_t idx = ((size_t)s * N + i) * 3 + a;
                    c->F[idx] = -(c->mass[i] * w2) * c->q[idx];
                }
    } else {
        int nthreads = 1;
#ifdef _OPENMP
        nthreads = omp_get_max_threads();
#endif
        g_inner_parallel = (nsys < nthreads);
        int64_t cap = sys_pair_cap(c);
        /* cap the per-system list at a density-based bound for large N to keep memory sane */
        if (c->periodic) {
            double vol = c->box[0] * c->box[1] * c->box[2];
            double expect = (double)N / vol * 4.18879020478639 * c->net.r_cut * c->net.r_cut * c->net.r_cut;
            int64_t cap2 = (int64_t)(N * (4.0 * expect + 64.0));
            if (cap2 < cap) cap = cap2;
        }
#pragma omp parallel for schedule(dynamic) if (!g_inner_parallel)
        for (int s = 0; s < nsys; ++s) {
            int32_t *rp = (int32_t *)malloc(sizeof(int32_t) * (N + 1));
            int32_t *cl = (int32_t *)malloc(sizeof(int32_t) * (size_t)cap);
            const double *qs = c->q + (size_t)s * N * 3;
            /* step 4 of N3: rebuild the list */
            if (ref_nlist_cell(N, qs, c->box, c->net.r_cut, rp, cl, cap) < 0) {
#pragma omp atomic write
                overflow = 1;
            } else {
                gfn_forces_system(c, qs, rp, cl, c->F + (size_t)s * N * 3, c->Fgross ? c->Fgross + (size_t)s * N : NULL);
            }
            free(rp); free(cl);
        }
    }
    if (c->md_cv) metad_add_bias_forces(c);
    c->forces_valid = 1;
    return overflow ? -3 : 0;
}

/* ------------------------------------------------------------------ */
/* integrator (N1-N5)                                                   */
/* ------------------------------------------------------------------ */
static inline size_t idx4(const ref_ctx *c, int r, int k, int i, int a)
{
    return ((((size_t)r * c->P + k) * c->N + i) * 3) + a;
}

/* v~_k = sum_j C_jk v_j for one (r, i, a) column */
static void to_modes(const ref_ctx *c, const double *v, int r, int i, int a, double *vt)
{
    for (int k = 0; k < c->P; ++k) {
        double s = 0.0;
        for (int j = 0; j < c->P; ++j) s += c->C[j * c->P + k] * v[idx4(c, r, j, i, a)];
        vt[k] = s;
    }
}
/* v_j = sum_k C_jk v~_k */
static void from_modes(const ref_ctx *c, const double *vt, int r, int i, int a, double *v)
{
    for (int j = 0; j < c->P; ++j) {
        double s = 0.0;
        for (int k = 0; k < c->P; ++k) s += c->C[j * c->P + k] * vt[k];
        v[idx4(c, r, j, i, a)] = s;
    }
}

static double beta_P(const ref_ctx *c) { return 1.0 / (KB_EV * c->T * c->P); }

/* O(dt/2): PILE-L in mode space (N3.1) */
static void step_O(ref_ctx *c, uint32_t t, uint32_t tag)
{
    const int P = c->P;
    const double bP = beta_P(c), hdt = 0.5 * c->dt;
#pragma omp parallel for collapse(2) schedule(static)
    for (int r = 0; r < c->R; ++r)
        for (int i = 0; i < c->N; ++i) {
            double pt[3][1024];
            for (int a = 0; a < 3; ++a) to_modes(c, c->p, r, i, a, pt[a]);
            for (int k = 0; k < P; ++k) {
                double gam = (k == 0) ? c->gamma_fs : 2.0 * c->omega_k[k];
                double c1 = exp(-gam * hdt), c2 = sqrt(1.0 - c1 * c1);
                double xi[3];
                ref_normal3(c->seed, (uint32_t)i, (uint32_t)(r * P + k), t, tag, xi);
                double sig = sqrt(c->mass[i] / bP);
                for (int a = 0; a < 3; ++a) pt[a][k] = c1 * pt[a][k] + sig * c2 * xi[a];
            }
            for (int a = 0; a < 3; ++a) from_modes(c, pt[a], r, i, a, c->p);
        }
}

/* B(dt/2): p += dt/2 F */
static void step_B(ref_ctx *c)
{
    size_t n = (size_t)c->R * c->P * c->N * 3;
    double hdt = 0.5 * c->dt;
    for (size_t t = 0; t < n; ++t) c->p[t] += hdt * c->F[t];
}

/* A(dt): exact free ring-polymer propagation in normal modes (N3.3) */
static void step_A(ref_ctx *c)
{
    const int P = c->P;
    const double dt = c->dt;
#pragma omp parallel for collapse(2) schedule(static)
    for (int r = 0; r < c->R; ++r)
        for (int i = 0; i < c->N; ++i) {
            double mi = c->mass[i];
            for (int a = 0; a < 3; ++a) {
                double qt[1024], pt[1024];
                to_modes(c, c->q, r, i, a, qt);
                to_modes(c, c->p, r, i, a, pt);
                for (int k = 0; k < P; ++k) {
                    if (k == 0) {
                        qt[0] = qt[0] + dt * pt[0] / mi;
                    } else {
                        double w = c->omega_k[k], cs = cos(w * dt), sn = sin(w * dt);
                        double pn = cs * pt[k] - mi * w * sn * qt[k];
                        double qn = sn / (mi * w) * pt[k] + cs * qt[k];
                        pt[k] = pn; qt[k] = qn;
                    }
                }
                from_modes(c, qt, r, i, a, c->q);
                from_modes(c, pt, r, i, a, c->p);
            }
        }
}


/* ------------------------------------------------------------------ */
/* integrator variants: staging transformation, PILE-G, primitive                                   */
/* P:L52 "the normal mode or staging transformation is employed to decouple the evolution of individual beads";    */
/* P:L114 "For primitive PIMD, inter-bead harmonic coupling potentials are incorporated as pluggable energy terms" */
/* ------------------------------------------------------------------ */
/* Staging variables (Tuckerman, Berne, Martyna, Klein 1993), beads j = 0..P-1 with q_P = q_0:
 *   u_0 = q_0,   u_j = q_j - (j q_{j+1} + q_0) / (j + 1)   for j = 1..P-1
 * Staging masses: lam_0 = 1 (no spring), lam_j = (j+1)/j for j >= 1, so that
 *   sum_j 1/2 m w_P^2 (q_j - q_{j+1})^2 = sum_{j>=1} 1/2 m lam_j w_P^2 u_j^2,
 * and with kinetic masses m lam_j every staging mode j >= 1 oscillates at w_P; u_0 moves freely with mass m.   */
static void stage_fwd(const double *q, double *u, int P)
{
    u[0] = q[0];
    for (int j = 1; j < P; ++j) {
        double qn = (j + 1 < P) ? q[j + 1] : q[0];
        u[j] = q[j] - ((double)j * qn + q[0]) / (double)(j + 1);
    }
}
/* inverse, from the top bead down: q_0 = u_0; q_j = u_j + j/(j+1) q_{j+1} + u_0/(j+1) */
static void stage_inv(const double *u, double *q, int P)
{
    q[0] = u[0];
    for (int j = P - 1; j >= 1; --j) {
        double qn = (j + 1 < P) ? q[j + 1] : q[0];
        q[j] = u[j] + ((double)j / (double)(j + 1)) * qn + u[0] / (double)(j + 1);
    }
}
/* chain rule dV/du from dV/dq (the same map takes bead momenta p_q to staging momenta p_u):
 *   f_u0 = sum_j f_qj;   f_uj = f_qj + (j-1)/j f_u(j-1)  for j >= 1 */
static void stage_force(const double *fq, double *fu, int P)
{
    double s = 0.0;
    for (int j = 0; j < P; ++j) s += fq[j];
    fu[0] = s;
    for (int j = 1; j < P; ++j) fu[j] = fq[j] + ((j > 1) ? ((double)(j - 1) / (double)j) * fu[j - 1] : 0.0);
}
/* canonical bead momenta from staging momenta, p_qj = sum_k (du_k/dq_j) p_uk, read off the definition of u:
 *   p_q0 = p_u0 - sum_{k>=1} p_uk/(k+1) - (P-1)/P p_u(P-1)   (the last term: q_P = q_0 inside u_{P-1}; P >= 2)
 *   p_qj = p_uj - (j-1)/j p_u(j-1)                            for j >= 1 */
static void stage_mom_to_bead(const double *pu, double *pq, int P)
{
    double s = pu[0];
    for (int k = 1; k < P; ++k) s -= pu[k] / (double)(k + 1);
    if (P >= 2) s -= ((double)(P - 1) / (double)P) * pu[P - 1];
    pq[0] = s;
    for (int j = 1; j < P; ++j) pq[j] = pu[j] - ((j > 1) ? ((double)(j - 1) / (double)j) * pu[j - 1] : 0.0);
}
static double stage_lam(int j) { return j == 0 ? 1.0 : (double)(j + 1) / (double)j; }

/* gather / scatter one (r, i, a) column of P beads */
static void col_get(const ref_ctx *c, const double *v, int r, int i, int a, double *out)
{
    for (int j = 0; j < c->P; ++j) out[j] = v[idx4(c, r, j, i, a)];
}
static void col_put(const ref_ctx *c, double *v, int r, int i, int a, const double *in)
{
    for (int j = 0; j < c->P; ++j) v[idx4(c, r, j, i, a)] = in[j];
}

/* The state array p always holds canonical BEAD momenta p_q (conjugate to q).  Mode momenta of one column: */
static void mom_to_modes(const ref_ctx *c, int r, int i, int a, double *pm)
{
    double pq[1024];
    if (c->transform == 0) { to_modes(c, c->p, r, i, a, pm); return; }
    col_get(c, c->p, r, i, a, pq);
    if (c->transform == 1) stage_force(pq, pm, c->P);
    else memcpy(pm, pq, sizeof(double) * c->P);
}
static void mom_from_modes(ref_ctx *c, int r, int i, int a, const double *pm)
{
    double pq[1024];
    if (c->transform == 0) { from_modes(c, pm, r, i, a, c->p); return; }
    if (c->transform == 1) stage_mom_to_bead(pm, pq, c->P);
    else memcpy(pq, pm, sizeof(double) * c->P);
    col_put(c, c->p, r, i, a, pq);
}
/* mass factor, free-ring frequency and PILE friction of mode k */
static double mode_lam(const ref_ctx *c, int k) { return c->transform == 1 ? stage_lam(k) : 1.0; }
static double mode_omega(const ref_ctx *c, int k)
{
    if (c->transform == 0) return c->omega_k[k];
    if (c->transform == 1) return k == 0 ? 0.0 : c->P * KB_EV * c->T / HBAR_EVFS;
    return 0.0; /* primitive: springs are explicit forces, every bead flies freely in A */
}
static double mode_gamma(const ref_ctx *c, int k)
{
    if (c->transform == 2) return c->gamma_fs; /* white-noise Langevin on every bead */
    return (k == 0) ? c->gamma_fs : 2.0 * mode_omega(c, k); /* PILE: critical damping of the free-ring mode */
}

/* O(dt/2) for any transform / thermostat.  PILE-G (Ceriotti, Parrinello, Markland, Manolopoulos 2010, sec. II.D with the
 * stochastic velocity rescaling of Bussi, Donadio, Parrinello 2007): the free mode (k = 0) of ALL atoms of a replica is scaled by
 *   alpha^2 = c + (1-c) (R1^2 + S) / (2 beta_P K) + 2 R1 sqrt(c (1-c) / (2 beta_P K)),   c = exp(-gamma dt/2),
 *   sign(alpha) = sign(R1 + sqrt(2 beta_P K c / (1-c))),
 * K = kinetic energy of the free modes, R1 and S = the first normal and the sum of the squares of the other 3N-1 normals
 * of the SAME counter-based stream PILE-L would use for mode 0 (atom, r*P+0, step, tag): R1 = (atom 0, x). */
static void step_O_general(ref_ctx *c, uint32_t t, uint32_t tag)
{
    const int P = c->P;
    const double bP = beta_P(c), hdt = 0.5 * c->dt;
    for (int r = 0; r < c->R; ++r) {
        double alpha = 1.0;
        if (c->thermostat == 1) {
            double K = 0.0, R1 = 0.0, S = 0.0;
            for (int i = 0; i < c->N; ++i) {
                double xi[3];
                ref_normal3(c->seed, (uint32_t)i, (uint32_t)(r * P + 0), t, tag, xi);
                for (int a = 0; a < 3; ++a) {
                    double pm[1024];
                    mom_to_modes(c, r, i, a, pm);
                    K += pm[0] * pm[0] / (2.0 * c->mass[i] * mode_lam(c, 0));
                    if (i == 0 && a == 0) R1 = xi[a]; else S += xi[a] * xi[a];
                }
            }
            double c1 = exp(-c->gamma_fs * hdt);
            if (K > 0.0) {
                double a2 = c1 + (1.0 - c1) * (R1 * R1 + S) / (2.0 * bP * K) + 2.0 * R1 * sqrt(c1 * (1.0 - c1) / (2.0 * bP * K));
                double sgn = (R1 + sqrt(2.0 * bP * K * c1 / (1.0 - c1)) >= 0.0) ? 1.0 : -1.0;
                alpha = sgn * sqrt(a2 > 0.0 ? a2 : 0.0);
            }
        }
#pragma omp parallel for schedule(static)
        for (int i = 0; i < c->N; ++i) {
            for (int a = 0; a < 3; ++a) {
                double pm[1024];
                mom_to_modes(c, r, i, a, pm);
                for (int k = 0; k < P; ++k) {
                    if (k == 0 && c->thermostat == 1) { pm[0] *= alpha; continue; }
                    double gam = mode_gamma(c, k);
                    double c1 = exp(-gam * hdt), c2 = sqrt(1.0 - c1 * c1);
                    double xi[3];
                    ref_normal3(c->seed, (uint32_t)i, (uint32_t)(r * P + k), t, tag, xi);
                    pm[k] = c1 * pm[k] + sqrt(c->mass[i] * mode_lam(c, k) / bP) * c2 * xi[a];
                }
                mom_from_modes(c, r, i, a, pm);
            }
        }
    }
}

/* B(dt/2) for the primitive variant: physical force plus the explicit ring springs -m w_P^2 (2 q_j - q_{j-1} - q_{j+1}) */
static void step_B_primitive(ref_ctx *c)
{
    const int P = c->P;
    const double hdt = 0.5 * c->dt, wP = P * KB_EV * c->T / HBAR_EVFS;
    for (int r = 0; r < c->R; ++r)
        for (int i = 0; i < c->N; ++i)
            for (int a = 0; a < 3; ++a)
                for (int j = 0; j < P; ++j) {
                    double qj = c->q[idx4(c, r, j, i, a)];
                    double qm = c->q[idx4(c, r, (j + P - 1) % P, i, a)], qp = c->q[idx4(c, r, (j + 1) % P, i, a)];
                    double fs = -c->mass[i] * wP * wP * ((qj - qm) + (qj - qp));
                    c->p[idx4(c, r, j, i, a)] += hdt * (c->F[idx4(c, r, j, i, a)] + fs);
                }
}

/* A(dt): exact propagation of every mode under its own free-ring Hamiltonian p^2/(2 m lam) + 1/2 m lam w^2 u^2 */
static void step_A_general(ref_ctx *c)
{
    const int P = c->P;
    const double dt = c->dt;
#pragma omp parallel for collapse(2) schedule(static)
    for (int r = 0; r < c->R; ++r)
        for (int i = 0; i < c->N; ++i)
            for (int a = 0; a < 3; ++a) {
                double qb[1024], um[1024], pm[1024];
                col_get(c, c->q, r, i, a, qb);
                if (c->transform == 0) to_modes(c, c->q, r, i, a, um);
                else if (c->transform == 1) stage_fwd(qb, um, P);
                else memcpy(um, qb, sizeof(double) * P);
                mom_to_modes(c, r, i, a, pm);
                for (int k = 0; k < P; ++k) {
                    double mu = c->mass[i] * mode_lam(c, k), w = mode_omega(c, k);
                    if (w == 0.0) {
                        um[k] = um[k] + dt * pm[k] / mu;
                    } else {
                        double cs = cos(w * dt), sn = sin(w * dt);
                        double pn = cs * pm[k] - mu * w * sn * um[k];
                        double un = sn / (mu * w) * pm[k] + cs * um[k];
                        pm[k] = pn; um[k] = un;
                    }
                }
                if (c->transform == 0) from_modes(c, um, r, i, a, c->q);
                else {
                    if (c->transform == 1) stage_inv(um, qb, P); else memcpy(qb, um, sizeof(double) * P);
                    col_put(c, c->q, r, i, a, qb);
                }
                mom_from_modes(c, r, i, a, pm);
            }
}

/* N5 in the chosen representation: mode momenta ~ N(0, m lam_k / beta_P), tag 2 */
static void init_momenta_general(ref_ctx *c)
{
    const double bP = beta_P(c);
    for (int r = 0; r < c->R; ++r)
        for (int i = 0; i < c->N; ++i) {
            double pm[3][1024];
            for (int k = 0; k < c->P; ++k) {
                double xi[3];
                ref_normal3(c->seed, (uint32_t)i, (uint32_t)(r * c->P + k), 0u, 2u, xi);
                for (int a = 0; a < 3; ++a) pm[a][k] = sqrt(c->mass[i] * mode_lam(c, k) / bP) * xi[a];
            }
            for (int a = 0; a < 3; ++a) mom_from_modes(c, r, i, a, pm[a]);
        }
}

/* Choose the integrator variant; to be called before the first step (it redraws the initial momenta, N5). */
int ref_set_integrator(ref_ctx *c, int transform, int thermostat)
{
    if (!c || transform < 0 || transform > 2 || thermostat < 0 || thermostat > 1 || c->step != 0) return -1;
    if (thermostat == 1 && transform == 2) return -1; /* PILE-G needs a free (centroid-like) mode */
    c->transform = transform; c->thermostat = thermostat;
    init_momenta_general(c);
    return 0;
}

int ref_step(ref_ctx *c, int n)
{
    if (!c || n < 0) return -1;
    if (c->P > 1024) return -1;
    int rc = 0;
    if (!c->forces_valid) rc = compute_forces(c);
    if (rc) return rc;
    for (int s = 0; s < n; ++s) {
        uint32_t t = (uint32_t)c->step;
        if (c->transform == 0 && c->thermostat == 0) { /* N3: normal modes + PILE-L */
            if (c->gamma_fs >= 0.0) step_O(c, t, 0u);
            step_B(c);
            step_A(c);
            rc = compute_forces(c);
            if (rc) return rc;
            step_B(c);
            if (c->gamma_fs >= 0.0) step_O(c, t, 1u);
        } else { /* same O B A [forces] B O splitting, other representation / thermostat (8(f)4) */
            if (c->gamma_fs >= 0.0) step_O_general(c, t, 0u);
            if (c->transform == 2) step_B_primitive(c); else step_B(c);
            step_A_general(c);
            rc = compute_forces(c);
            if (rc) return rc;
            if (c->transform == 2) step_B_primitive(c); else step_B(c);
            if (c->gamma_fs >= 0.0) step_O_general(c, t, 1u);
        }
        c->step += 1;
        if (c->md_cv && c->md_every > 0 && c->step % c->md_every == 0) {
            /* the Gaussians go in at the positions reached by this step; the forces F(q) of the state include them from here on */
            metad_deposit(c);
            rc = compute_forces(c);
            if (rc) return rc;
        }
    }
    return 0;
}

/* ------------------------------------------------------------------ */
/* create / destroy / accessors                                         */
/* ------------------------------------------------------------------ */
static double *take_T(const float **w, int n_out, int n_in)
{ /* read a row-major [out][in] fp32 matrix, return fp64 [in][out] */
    double *t = (double *)malloc(sizeof(double) * (size_t)n_out * n_in);
    for (int o = 0; o < n_out; ++o)
        for (int k = 0; k < n_in; ++k) t[(size_t)k * n_out + o] = (double)(*w)[(size_t)o * n_in + k];
    *w += (size_t)n_out * n_in;
    return t;
}
static double *take_v(const float **w, int n)
{
    double *t = (double *)malloc(sizeof(double) * (size_t)n);
    for (int o = 0; o < n; ++o) t[o] = (double)(*w)[o];
    *w += n;
    return t;
}

int64_t ref_n_weights(int S, int K, int H, int L)
{
    return (int64_t)S * H + (int64_t)H * K + H + (int64_t)H * H + H + (int64_t)L * (5LL * H * H + 3LL * H) + (int64_t)H * H +
           H + H + 1;
}

void ref_destroy(ref_ctx *c);

int ref_create(ref_ctx **out, int n_atoms, int n_replicas, const int32_t *species, const double *masses_amu,
               const double *positions, const double box[3], int P, double T_kelvin, double dt_fs,
               double gamma_centroid_per_ps, uint64_t seed, const ref_net_params *net)
{
    if (!out || n_atoms < 1 || n_replicas < 1 || P < 1 || P > 1024 || !species || !masses_amu || !positions || !net)
        return -1;
    if (!(T_kelvin > 0.0) || !(dt_fs > 0.0)) return -1;
    int periodic = box[0] > 0.0 || box[1] > 0.0 || box[2] > 0.0;
    if (periodic && !(box[0] > 0.0 && box[1] > 0.0 && box[2] > 0.0)) return -1;
    if (net->kind == 0) {
        if (net->hidden > 512 || net->n_rbf > 512 || net->n_rbf < 2) return -1;
        if (net->n_weights != ref_n_weights(net->n_species, net->n_rbf, net->hidden, net->n_layers)) return -1;
        if (periodic)
            for (int a = 0; a < 3; ++a)
                if (box[a] < 2.0 * net->r_cut) return -1; /* L4 */
    }
    ref_ctx *c = (ref_ctx *)calloc(1, sizeof(ref_ctx));
    c->N = n_atoms; c->R = n_replicas; c->P = P; c->periodic = periodic;
    for (int a = 0; a < 3; ++a) c->box[a] = box[a];
    c->T = T_kelvin; c->dt = dt_fs; c->gamma_fs = gamma_centroid_per_ps < 0.0 ? -1.0 : gamma_centroid_per_ps * 1e-3;
    c->seed = seed; c->step = 0; c->net = *net;
    c->species = (int32_t *)malloc(sizeof(int32_t) * n_atoms);
    c->mass = (double *)malloc(sizeof(double) * n_atoms);
    for (int i = 0; i < n_atoms; ++i) {
        c->species[i] = species[i];
        c->mass[i] = masses_amu[species[i]] * AMU_INTERNAL;
    }
    if (net->kind == 0) {
        const int S = net->n_species, K = net->n_rbf, H = net->hidden, L = net->n_layers;
        const float *w = net->weights;
        c->Emb = take_v(&w, S * H); /* [S][H], used row-wise */
        c->We1 = take_T(&w, H, K); c->be1 = take_v(&w, H);
        c->We2 = take_T(&w, H, H); c->be2 = take_v(&w, H);
        c->Ws = (double **)calloc(L, sizeof(double *)); c->Wvn = (double **)calloc(L, sizeof(double *));
        c->Wvm = (double **)calloc(L, sizeof(double *)); c->bv1 = (double **)calloc(L, sizeof(double *));
        c->Wv2 = (double **)calloc(L, sizeof(double *)); c->bv2 = (double **)calloc(L, sizeof(double *));
        c->Wa = (double **)calloc(L, sizeof(double *)); c->ba = (double **)calloc(L, sizeof(double *));
        for (int l = 0; l < L; ++l) {
            c->Ws[l] = take_T(&w, H, H); c->Wvn[l] = take_T(&w, H, H); c->Wvm[l] = take_T(&w, H, H);
            c->bv1[l] = take_v(&w, H); c->Wv2[l] = take_T(&w, H, H); c->bv2[l] = take_v(&w, H);
            c->Wa[l] = take_T(&w, H, H); c->ba[l] = take_v(&w, H);
        }
        c->Wf1 = take_T(&w, H, H); c->bf1 = take_v(&w, H); c->wf2 = take_v(&w, H);
        c->bf2 = (double)*w;
        c->net.weights = NULL;
    }
    size_t n = (size_t)c->R * P * n_atoms * 3;
    c->q = (double *)malloc(sizeof(double) * n);
    c->p = (double *)malloc(sizeof(double) * n);
    c->F = (double *)calloc(n, sizeof(double));
    c->Fgross = (double *)calloc(n / 3 + 1, sizeof(double));
    c->C = (double *)malloc(sizeof(double) * (size_t)P * P);
    c->omega_k = (double *)malloc(sizeof(double) * P);
    ref_nm_matrix(P, c->C);
    const double pi = 3.14159265358979323846264338327950288;
    double omega_P = P * KB_EV * T_kelvin / HBAR_EVFS; /* N1 */
    for (int k = 0; k < P; ++k) c->omega_k[k] = 2.0 * omega_P * sin(k * pi / P);
    /* N5: all beads on the input geometry; momenta drawn per mode with tag 2, t = 0 */
    for (int r = 0; r < c->R; ++r)
        for (int k = 0; k < P; ++k)
            for (int i = 0; i < n_atoms; ++i)
                for (int a = 0; a < 3; ++a) c->q[idx4(c, r, k, i, a)] = positions[((size_t)r * n_atoms + i) * 3 + a];
    double bP = beta_P(c);
    for (int r = 0; r < c->R; ++r)
        for (int i = 0; i < n_atoms; ++i) {
            double pt[3][1024];
            for (int k = 0; k < P; ++k) {
                double xi[3];
                ref_normal3(seed, (uint32_t)i, (uint32_t)(r * P + k), 0u, 2u, xi);
                for (int a = 0; a < 3; ++a) pt[a][k] = sqrt(c->mass[i] / bP) * xi[a];
            }
            for (int a = 0; a < 3; ++a) from_modes(c, pt[a], r, i, a, c->p);
        }
    c->forces_valid = 0;
    *out = c;
    return 0;
}

void ref_destroy(ref_ctx *c)
{
    if (!c) return;
    free(c->species); free(c->mass); free(c->q); free(c->p); free(c->F); free(c->Fgross); free(c->C); free(c->omega_k);
    free(c->md_n); free(c->md_c); free(c->md_h); free(c->md_s); free(c->md_ds);
    if (c->net.kind == 0) {
        free(c->Emb); free(c->We1); free(c->be1); free(c->We2); free(c->be2);
        for (int l = 0; l < c->net.n_layers; ++l) {
            free(c->Ws[l]); free(c->Wvn[l]); free(c->Wvm[l]); free(c->bv1[l]);
            free(c->Wv2[l]); free(c->bv2[l]); free(c->Wa[l]); free(c->ba[l]);
        }
        free(c->Ws); free(c->Wvn); free(c->Wvm); free(c->bv1); free(c->Wv2); free(c->bv2); free(c->Wa); free(c->ba);
        free(c->Wf1); free(c->bf1); free(c->wf2);
    }
    free(c);
}

int ref_forces(ref_ctx *c, double *out)
{ /* [R][P][N][3] eV/A, recomputed at the current q */
    if (!c || !out) return -1;
    int rc = compute_forces(c);
    if (rc) return rc;
    memcpy(out, c->F, sizeof(double) * (size_t)c->R * c->P * c->N * 3);
    return 0;
}

int ref_force_gross(ref_ctx *c, double *out)
{ /* [R][P][N]: sum of the magnitudes of the terms of F_i at the current q (diagnostic scale for error bounds; kind 0) */
    if (!c || !out || c->net.kind != 0) return -1;
    int rc = compute_forces(c);
    if (rc) return rc;
    memcpy(out, c->Fgross, sizeof(double) * (size_t)c->R * c->P * c->N);
    return 0;
}

int ref_get_state(ref_ctx *c, double *q, double *p, int64_t *step)
{
    size_t n = (size_t)c->R * c->P * c->N * 3;
    if (q) memcpy(q, c->q, sizeof(double) * n);
    if (p) memcpy(p, c->p, sizeof(double) * n);
    if (step) *step = c->step;
    return 0;
}

int ref_set_state(ref_ctx *c, const double *q, const double *p, int64_t step)
{
    size_t n = (size_t)c->R * c->P * c->N * 3;
    if (q) memcpy(c->q, q, sizeof(double) * n);
    if (p) memcpy(c->p, p, sizeof(double) * n);
    c->step = step;
    c->forces_valid = 0;
    return 0;
}

/* global CSR over all rows (row id = (r*P + k)*N + i); col holds the atom index j within the bead-system */
int ref_nlist(ref_ctx *c, int32_t *row_ptr, int32_t *col, int64_t col_capacity, int64_t *n_pairs, int use_brute)
{
    const int N = c->N, nsys = c->R * c->P;
    int64_t total = 0;
    int32_t *rp = (int32_t *)malloc(sizeof(int32_t) * (N + 1));
    for (int s = 0; s < nsys; ++s) {
        const double *qs = c->q + (size_t)s * N * 3;
        int64_t n = use_brute ? ref_nlist_brute(N, qs, c->box, c->net.r_cut, rp, col + total, col_capacity - total)
                              : ref_nlist_cell(N, qs, c->box, c->net.r_cut, rp, col + total, col_capacity - total);
        if (n < 0) { free(rp); return -3; }
        for (int i = 0; i < N; ++i) row_ptr[(size_t)s * N + i] = (int32_t)(total + rp[i]);
        total += n;
    }
    row_ptr[(size_t)nsys * N] = (int32_t)total;
    if (n_pairs) *n_pairs = total;
    free(rp);
    return 0;
}

/* estimators E1-E4 + centroid temperature, per replica (P:L56-58 bead average) */
int ref_estimators(ref_ctx *c, ref_estimators_t *out)
{
    if (!c || !out) return -1;
    if (!c->forces_valid) compute_forces(c);
    const int N = c->N, P = c->P;
    const double kT = KB_EV * c->T;
    double omega_P = P * kT / HBAR_EVFS;
    for (int r = 0; r < c->R; ++r) {
        double spring = 0.0, vir = 0.0, cvir = 0.0, vpot = 0.0, tc = 0.0;
        for (int i = 0; i < N; ++i) {
            double qbar[3] = {0, 0, 0}, pc[3] = {0, 0, 0};
            for (int k = 0; k < P; ++k)
                for (int a = 0; a < 3; ++a) {
                    qbar[a] += c->q[idx4(c, r, k, i, a)];
                    /* momentum of the free mode: p~_0 = sum_j p_j / sqrt(P) (normal modes; same normalisation for primitive),
                       p_u0 = sum_j p_j (staging, whose free mode has mass m instead of the ring's P m / P) */
                    pc[a] += (c->transform == 1 ? 1.0 : c->C[k * P + 0]) * c->p[idx4(c, r, k, i, a)];
                }
            for (int a = 0; a < 3; ++a) qbar[a] /= P;
            for (int k = 0; k < P; ++k) {
                int kn = (k + 1) % P;
                for (int a = 0; a < 3; ++a) {
                    double qk = c->q[idx4(c, r, k, i, a)], dq = qk - c->q[idx4(c, r, kn, i, a)];
                    double f = c->F[idx4(c, r, k, i, a)];
                    spring += 0.5 * c->mass[i] * omega_P * omega_P * dq * dq;
                    vir += qk * f;
                    cvir += (qk - qbar[a]) * f;
                    if (c->net.kind == 1)
                        vpot += 0.5 * c->mass[i] * c->net.harmonic_omega * c->net.harmonic_omega * qk * qk;
                }
            }
            for (int a = 0; a < 3; ++a) tc += pc[a] * pc[a] / c->mass[i];
        }
        out[r].k_prim = 1.5 * N * P * kT - spring / P;
        out[r].k_vir = -vir / (2.0 * P);
        out[r].k_cvir = 1.5 * N * kT - cvir / (2.0 * P);
        out[r].v_pot = (c->net.kind == 0) ? NAN : vpot / P;
        out[r].t_centroid = tc / (3.0 * N * KB_EV * P);
    }
    return 0;
}

/* metadynamics API.  cv: 1 s_dimer (atoms6 = O1, H1, O2, O4, H2, O3), 2 Debye (f_species[S], Q).  Energies in eV. */
int ref_metad_enable(ref_ctx *c, int cv, const int32_t *atoms6, const double *f_species, double Q, double sigma, double height_eV,
                     double bias_factor, int deposit_every, int max_gaussians)
{
    if (!c || (cv != 1 && cv != 2) || !(sigma > 0.0) || !(bias_factor > 1.0) || deposit_every < 1 || max_gaussians < 1) return -1;
    if (cv == 1) { if (!atoms6) return -1; for (int k = 0; k < 6; ++k) { if (atoms6[k] < 0 || atoms6[k] >= c->N) return -1; c->md_atoms[k] = atoms6[k]; } }
    if (cv == 2) { if (!f_species || c->net.n_species > 16 || !(Q > 0.0)) return -1; for (int k = 0; k < c->net.n_species; ++k) c->md_f[k] = f_species[k]; c->md_Q = Q; }
    c->md_cv = cv; c->md_sigma = sigma; c->md_w0 = height_eV; c->md_biasf = bias_factor; c->md_every = deposit_every; c->md_max = max_gaussians;
    free(c->md_n); free(c->md_c); free(c->md_h); free(c->md_s); free(c->md_ds);
    c->md_n = (int *)calloc((size_t)c->R, sizeof(int));
    c->md_c = (double *)calloc((size_t)c->R * max_gaussians, sizeof(double));
    c->md_h = (double *)calloc((size_t)c->R * max_gaussians, sizeof(double));
    c->md_s = (double *)calloc((size_t)c->R * c->P, sizeof(double));
    c->md_ds = (double *)calloc((size_t)c->R * c->P * c->N * 3, sizeof(double));
    c->forces_valid = 0;
    return 0;
}
/* CV of every bead [R][P] and its gradient [R][P][N][3] at the current positions; either may be NULL */
int ref_metad_cv(ref_ctx *c, double *s_out, double *grad_out)
{
    if (!c || !c->md_cv) return -1;
    int rc = compute_forces(c);
    if (rc) return rc;
    if (s_out) memcpy(s_out, c->md_s, sizeof(double) * (size_t)c->R * c->P);
    if (grad_out) memcpy(grad_out, c->md_ds, sizeof(double) * (size_t)c->R * c->P * c->N * 3);
    return 0;
}
/* deposited Gaussians of replica r: count; centres and heights into caller arrays of capacity cap */
int ref_metad_gaussians(ref_ctx *c, int r, double *centres, double *heights, int cap)
{
    if (!c || !c->md_cv || r < 0 || r >= c->R) return -1;
    const int n = c->md_n[r];
    for (int g = 0; g < n && g < cap; ++g) { if (centres) centres[g] = c->md_c[(size_t)r * c->md_max + g]; if (heights) heights[g] = c->md_h[(size_t)r * c->md_max + g]; }
    return n;
}
/* bias energy V_G(s) of replica r at a given CV value */
double ref_metad_bias(ref_ctx *c, int r, double s) { return (c && c->md_cv && r >= 0 && r < c->R) ? md_bias(c, r, s, NULL) : 0.0; }
/* one deposition event now (tests) */
int ref_metad_deposit_now(ref_ctx *c)
{
    if (!c || !c->md_cv) return -1;
    int rc = c->forces_valid ? 0 : compute_forces(c);
    if (rc) return rc;
    metad_deposit(c);
    c->forces_valid = 0;
    return 0;
}

/* test access to the staging maps of one column (P values each) */
void ref_stage_fwd(const double *q, double *u, int P) { stage_fwd(q, u, P); }
void ref_stage_inv(const double *u, double *q, int P) { stage_inv(u, q, P); }
void ref_stage_force(const double *fq, double *fu, int P) { stage_force(fq, fu, P); }
void ref_stage_mom_to_bead(const double *pu, double *pq, int P) { stage_mom_to_bead(pu, pq, P); }

void ref_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

int ref_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
