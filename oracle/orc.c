/* oracle/orc.c -- CPU ORACLE, TEST INFRASTRUCTURE ONLY (see orc.h).
 *
 * Plain nested loops over cells, nodes and edges, in the paper's order and notation; fp64 by
 * default.  No blocking, fusion or layout tricks.  OpenMP over z-planes (cells), nodes and meshes
 * only ("It may use OpenMP over z-planes and over meshes; nothing else"): every
 * parallel loop runs the same per-cell / per-node / per-mesh body as the serial one; the spread adds
 * into the shared force field with `omp atomic`, so its sums are reordered at the 1e-16 level (any
 * summation order is correct there).
 * Every function cites the passage of /root/reference/PAPER.md it follows ("L" = line number)
 * or the SURVEY.md section 8(c) reading ("O-n", "G-n") taken where the paper is silent/garbled.
 *
 * PARITY UNPINNED (conventions fixed in DESIGN.md, not by the paper): which velocity is
 * interpolated (G11, reading A), the wall density rho_w = 1 (G9), dropped stencil cells at a
 * wall (G15), the corner rule for links leaving through two wall faces at once, closing the
 * on-site wall layers at initialisation (G25); for the adhesion model (NEXT-4): break-before-form
 * order within one update (A-5), lowest-receptor-index-first arbitration of the places of a vWF
 * site (A-7), nearest-site candidate (A-3), receptors sitting on mesh nodes (A-1); for the flipping
 * platelet (NEXT-3) the near-wall orbit (the paper's 2.65 % refers to a curve printed as an image).
 */
#include "orc.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>

#ifdef ORC_REAL_FLOAT
typedef float real;
#else
typedef double real;
#endif

#define Q 19
/* internal storage: the 19 values of a lattice site side by side (L181 "19 values f_i(x,t) are
 * stored at each lattice site"); the interface (orc.h) is SoA f[i*cells + q] */
#define FI(i, q) ((size_t)(q) * Q + (size_t)(i))
static const double PI = 3.14159265358979323846264338327950288;

/* D3Q19 vectors in the paper's numbering (1-based i -> row i-1).  The paper shows them only in
 * Fig. 4 (L434); the order is fixed uniquely by the boundary equations Eq. 23-30 (L217-238):
 * {i : c_z=+1} = {5,9,13,15,17}, opposites 5/6, 9/14, 13/10, 15/18, 17/16, +x set {1,7,8},
 * -x set {2,11,12}, +y set {3,7,11}, -y set {4,8,12}; rest population is i = 19 (Eq. 21).   */
static const int C[Q][3] = {
    {+1, 0, 0}, {-1, 0, 0}, {0, +1, 0}, {0, -1, 0}, {0, 0, +1}, {0, 0, -1},      /* 1..6   */
    {+1, +1, 0}, {+1, -1, 0}, {+1, 0, +1}, {+1, 0, -1},                           /* 7..10  */
    {-1, +1, 0}, {-1, -1, 0}, {-1, 0, +1}, {-1, 0, -1},                           /* 11..14 */
    {0, +1, +1}, {0, +1, -1}, {0, -1, +1}, {0, -1, -1},                           /* 15..18 */
    {0, 0, 0}};                                                                   /* 19     */

/* Eq. 21 (L208): 2/36 for i=1..6, 1/36 for i=7..18, 12/36 for i=19 */
static double weight(int i0) { return i0 < 6 ? 2.0 / 36.0 : (i0 < 18 ? 1.0 / 36.0 : 12.0 / 36.0); }

static int opposite(int i0) {
    for (int j = 0; j < Q; ++j)
        if (C[j][0] == -C[i0][0] && C[j][1] == -C[i0][1] && C[j][2] == -C[i0][2]) return j;
    return -1;
}
static int OPP[Q];   /* OPP[i] = opposite(i), filled by orc_create */

struct orc_ctx {
    int n[3];
    long cells;
    real tau;
    int kind[3];
    real u_lo[3][3], u_hi[3][3];
    real *f, *fstar, *g_last;          /* f[FI(i,q)]; g_last[d*cells+q] */
    /* meshes, concatenated in orc_add_mesh order */
    int n_nodes, n_edges, n_meshes, cap_nodes, cap_edges;
    real *X, *F, *U;                   /* AoS 3 per node */
    int *edge;                         /* global node index pairs */
    real *rest, *kspring;              /* per edge */
    /* NEXT-2 (Eq. 4-5): triangles of the lipid-bilayer surface, per mesh */
    int *mesh_off;                     /* first global node of mesh s (n_meshes + 1 entries) */
    int *mesh_edge_off;                /* first global edge of mesh s (n_meshes + 1 entries) */
    int n_tris, cap_tris;
    int *tri;                          /* global node index triples, outward orientation */
    int *tri_mesh;                     /* mesh of each triangle */
    real *tri_S0;                      /* unstressed triangle area S_0 */
    real *S0_tot, *V0, *k_s, *k_t, *k_v;   /* per mesh (k = 0 and no triangles until orc_set_triangles) */
    int forces_valid;
    /* NEXT-4 (section 3.2, 3.4.1): receptors, bonds to the vWF sites of one wall, wall repulsion */
    int n_rec;
    int *rec_node;                     /* global node each receptor sits on */
    int *bond;                         /* per receptor: (bound 0/1, site s0, site s1), sites unwrapped */
    int *site_count;                   /* bonds per vWF site, n[t0] * n[t1] */
    orc_adhesion adh;
};

void orc_lattice(int* c_out, double* w_out) {
    for (int i = 0; i < Q; ++i) {
        for (int d = 0; d < 3; ++d) c_out[3 * i + d] = C[i][d];
        w_out[i] = weight(i);
    }
}
int orc_real_bytes(void) { return (int)sizeof(real); }

/* ---- Eq. 36 (L273), with the second case read as |r| >= 2 (G6) -------------------------- */
double orc_phi(double r) {
    double a = fabs(r);
    if (a >= 2.0) return 0.0;
    return 0.25 * (1.0 + cos(PI * r / 2.0));
}
static real phi(real r) { return (real)orc_phi((double)r); }

/* ---- Eq. 20 (L203): f_eq = w rho [1 + c.v/cs^2 + (c.v)^2/(2 cs^4) - v^2/(2 cs^2)], cs^2 = 1/3 */
static real feq(int i, real rho, const real v[3]) {
    real cv = C[i][0] * v[0] + C[i][1] * v[1] + C[i][2] * v[2];
    real vv = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
    return (real)weight(i) * rho * ((real)1 + (real)3 * cv + (real)4.5 * cv * cv - (real)1.5 * vv);
}
double orc_feq(int i0, double rho, const double v[3]) {
    real vr[3] = {(real)v[0], (real)v[1], (real)v[2]};
    return (double)feq(i0, (real)rho, vr);
}

/* ---- O-8: Philox4x32-10 (Salmon et al., SC'11): 10 rounds of
 *   (c0,c1,c2,c3) <- (hi(M1 c2)^c1^k0, lo(M1 c2), hi(M0 c0)^c3^k1, lo(M0 c0)),
 * key bumped by the Weyl constants (W0, W1) between rounds.                                */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        if (r > 0) { k0 += W0; k1 += W1; }
        uint64_t p0 = (uint64_t)M0 * c0, p1 = (uint64_t)M1 * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}
/* xi = ((r >> 8) + 0.5) 2^-24: exact in fp32, never 0 or 1 */
double orc_uniform01(uint32_t r) { return ((double)(r >> 8) + 0.5) * (1.0 / 16777216.0); }

static void noise_words(uint64_t seed, uint64_t index, uint32_t step, uint32_t tag, uint32_t r[4]) {
    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    uint32_t ctr[4] = {(uint32_t)index, (uint32_t)(index >> 32), step, tag};
    orc_philox4x32_10(ctr, key, r);
}
void orc_noise_uniform(uint64_t seed, uint64_t index, uint32_t step, uint32_t tag, double xi[4]) {
    uint32_t r[4];
    noise_words(seed, index, step, tag, r);
    for (int j = 0; j < 4; ++j) xi[j] = orc_uniform01(r[j]);
}
/* Box-Muller: z0 = sqrt(-2 ln xi0) cos(2 pi xi1), z1 = same radius * sin(2 pi xi1),
 *             z2 = sqrt(-2 ln xi2) cos(2 pi xi3)                                            */
void orc_noise_normal3(uint64_t seed, uint64_t index, uint32_t step, uint32_t tag, double z[3]) {
    double xi[4];
    orc_noise_uniform(seed, index, step, tag, xi);
    double r0 = sqrt(-2.0 * log(xi[0])), r2 = sqrt(-2.0 * log(xi[2]));
    z[0] = r0 * cos(2.0 * PI * xi[1]);
    z[1] = r0 * sin(2.0 * PI * xi[1]);
    z[2] = r2 * cos(2.0 * PI * xi[3]);
}

/* the same for n indices at once (z: n x 3) -- a loop over the call above, for the tests */
void orc_noise_normal3_many(uint64_t seed, const uint64_t* index, long n, uint32_t step, uint32_t tag, double* z) {
#pragma omp parallel for schedule(static)
    for (long t = 0; t < n; ++t) orc_noise_normal3(seed, index[t], step, tag, z + 3 * t);
}

/* ------------------------------------------------------------------------------------------ */
int orc_create(int nx, int ny, int nz, double tau, const int kind[3], const double u_lo[9],
               const double u_hi[9], orc_ctx** out) {
    if (!out || nx < 1 || ny < 1 || nz < 1 || !(tau > 0.5) || !kind) return -1;
    orc_ctx* c = (orc_ctx*)calloc(1, sizeof(orc_ctx));
    for (int i = 0; i < Q; ++i) OPP[i] = opposite(i);
    c->n[0] = nx; c->n[1] = ny; c->n[2] = nz;
    c->cells = (long)nx * ny * nz;
    c->tau = (real)tau;
    for (int a = 0; a < 3; ++a) {
        if (kind[a] != ORC_PERIODIC && kind[a] != ORC_WALL && kind[a] != ORC_WALL_HH) { free(c); return -1; }
        /* NEXT-1: the on-site condition is written for a plane (L217); edges and corners where
         * two closed axes meet are not defined by the paper -> the other two axes must be periodic */
        if (kind[a] == ORC_WALL_HH && (a == 0 ? nx : a == 1 ? ny : nz) < 2) { free(c); return -1; }
        if (kind[a] == ORC_WALL_HH)
            for (int b = 0; b < 3; ++b)
                if (b != a && kind[b] != ORC_PERIODIC) { free(c); return -1; }
        c->kind[a] = kind[a];
        for (int d = 0; d < 3; ++d) {
            c->u_lo[a][d] = u_lo ? (real)u_lo[3 * a + d] : 0;
            c->u_hi[a][d] = u_hi ? (real)u_hi[3 * a + d] : 0;
        }
    }
    c->f = (real*)calloc((size_t)Q * c->cells, sizeof(real));
    c->fstar = (real*)calloc((size_t)Q * c->cells, sizeof(real));
    c->g_last = (real*)calloc((size_t)3 * c->cells, sizeof(real));
    if (!c->f || !c->fstar || !c->g_last) { orc_destroy(c); return -1; }
    *out = c;
    return 0;
}

int orc_destroy(orc_ctx* c) {
    if (!c) return -1;
    free(c->f); free(c->fstar); free(c->g_last);
    free(c->X); free(c->F); free(c->U); free(c->edge); free(c->rest); free(c->kspring);
    free(c->mesh_off); free(c->mesh_edge_off); free(c->tri); free(c->tri_mesh); free(c->tri_S0);
    free(c->S0_tot); free(c->V0); free(c->k_s); free(c->k_t); free(c->k_v);
    free(c->rec_node); free(c->bond); free(c->site_count);
    free(c);
    return 0;
}

static void hecht_harting_faces(orc_ctx* c);   /* NEXT-1, below */

/* O-2: f_i = feq_i(rho, u) (Eq. 20) + amp (2 xi - 1), xi = Philox uniform keyed on
 * (index = cell*19 + (i-1), step 0, tag 1), first output word. */
int orc_set_equilibrium(orc_ctx* c, const double* rho, const double* u, double amp, uint64_t seed) {
    if (!c) return -1;
    const long N = c->cells;
#pragma omp parallel for schedule(static)
    for (long q = 0; q < N; ++q) {
        real r = rho ? (real)rho[q] : (real)1;
        real v[3] = {u ? (real)u[q] : 0, u ? (real)u[N + q] : 0, u ? (real)u[2 * N + q] : 0};
        for (int i = 0; i < Q; ++i) {
            real val = feq(i, r, v);
            if (amp > 0) {
                double xi[4];
                orc_noise_uniform(seed, (uint64_t)q * Q + (uint64_t)i, 0u, 1u, xi);
                val += (real)(amp * (2.0 * xi[0] - 1.0));
            }
            c->f[FI(i, q)] = val;
        }
    }
    memset(c->g_last, 0, (size_t)3 * N * sizeof(real));
    hecht_harting_faces(c);
    return 0;
}

/* O-3 steps 1-5 for one cell: moments (Eq. 17-18), v = u + g/(2 rho) (L201), f_eq(rho, v)
 * (Eq. 20), BGK relaxation (Eq. 16) and the Guo term (Eq. 19 read per G3: the tensor
 * (c c^T - cs^2 I) and v, equivalent to S_i = (1 - 1/2tau) w_i [3 (c_i - v).g + 9 (c_i.v)(c_i.g)]). */
static void collide_cell(const orc_ctx* c, const real fin[Q], const real g[3], real fout[Q]) {
    real rho = 0, j[3] = {0, 0, 0};
    for (int i = 0; i < Q; ++i) {
        rho += fin[i];
        for (int d = 0; d < 3; ++d) j[d] += C[i][d] * fin[i];
    }
    real v[3];
    for (int d = 0; d < 3; ++d) v[d] = (j[d] + g[d] / 2) / rho;
    for (int i = 0; i < Q; ++i) {
        real cv = C[i][0] * v[0] + C[i][1] * v[1] + C[i][2] * v[2];
        real cg = C[i][0] * g[0] + C[i][1] * g[1] + C[i][2] * g[2];
        real cmv_g = (C[i][0] - v[0]) * g[0] + (C[i][1] - v[1]) * g[1] + (C[i][2] - v[2]) * g[2];
        real S = ((real)1 - (real)1 / (2 * c->tau)) * (real)weight(i) * ((real)3 * cmv_g + (real)9 * cv * cg);
        fout[i] = fin[i] - (fin[i] - feq(i, rho, v)) / c->tau + S;
    }
}

/* NEXT-1.  Hecht-Harting on-site velocity boundary (the paper's ref. [34]; Eq. 23-30).
 * The paper prints the plane z = 0 (inward normal n = +z): the populations with c.n = +1
 * (i = 5, 9, 13, 15, 17) are undetermined after streaming and, with the wall velocity v,
 *     rho  = [ sum_{c.n = 0} f_i + 2 sum_{c.n = -1} f_i ] / (1 - v.n)                 (first line of L219)
 *     f_5  = f_6  + rho v_z / 3
 *     f_9  = f_14 + rho (v_z + v_x)/6 - N_x     f_13 = f_10 + rho (v_z - v_x)/6 + N_x   (Eq. 25-26; "rho/eps" read rho/6, G5)
 *     f_15 = f_18 + rho (v_z + v_y)/6 - N_y     f_17 = f_16 + rho (v_z - v_y)/6 + N_y   (Eq. 27-28)
 *     N_t  = (1/2) [ sum_{c.n=0, c.t=+1} f_i - sum_{c.n=0, c.t=-1} f_i ] - rho v_t / 3   (Eq. 29-30)
 * Any other face is the same statement with the axes renamed: n = inward unit normal
 * (+e_a on the low face of axis a, -e_a on the high face), t runs over the two tangential axes,
 * and an unknown population with c = n + s t (s = +-1) is  f_opp + rho (v.n + s v_t)/6 - s N_t.
 * Paper-literal: the condition sets sum c_i f_i = rho v; a body force at the wall node enters
 * only through the usual g/2 of the collision and of lbm_read_macros (reading G24). */
static void hecht_harting_cell(real f[Q], int a, int face, const real vw[3]) {
    const int sgn = face ? -1 : +1;                     /* n = sgn e_a */
    const real vn = (real)sgn * vw[a];
    real S0 = 0, Sm = 0, T[3] = {0, 0, 0};
    for (int i = 0; i < Q; ++i) {
        const int cn = sgn * C[i][a];
        if (cn == 0) {
            S0 += f[i];
            for (int b = 0; b < 3; ++b) T[b] += C[i][b] * f[i];
        } else if (cn == -1) Sm += f[i];
    }
    const real rho = (S0 + 2 * Sm) / ((real)1 - vn);
    real N[3];
    for (int b = 0; b < 3; ++b) N[b] = T[b] / 2 - rho * vw[b] / 3;
    for (int i = 0; i < Q; ++i) {
        if (sgn * C[i][a] != 1) continue;
        int b = -1;
        for (int d = 0; d < 3; ++d)
            if (d != a && C[i][d] != 0) b = d;
        if (b < 0) f[i] = f[OPP[i]] + rho * vn / 3;
        else f[i] = f[OPP[i]] + rho * (vn + C[i][b] * vw[b]) / 6 - C[i][b] * N[b];
    }
}

/* NEXT-1: on an on-site velocity wall the populations pointing into the fluid do not arrive by
 * streaming ("undetermined", L217); they are filled from the others (Eq. 23-30) after every
 * streaming step -- and after lbm_set_equilibrium / lbm_write_populations, so that the stored
 * state always satisfies the wall condition (reading G25). */
static void hecht_harting_faces(orc_ctx* c) {
    const int nx = c->n[0], ny = c->n[1];
    for (int a = 0; a < 3; ++a) {
        if (c->kind[a] != ORC_WALL_HH) continue;
        for (int face = 0; face < 2; ++face) {
            const int b1 = (a + 1) % 3, b2 = (a + 2) % 3;
#pragma omp parallel for schedule(static)
            for (int s2 = 0; s2 < c->n[b2]; ++s2)
                for (int s1 = 0; s1 < c->n[b1]; ++s1) {
                    int xs[3];
                    xs[a] = face ? c->n[a] - 1 : 0;
                    xs[b1] = s1; xs[b2] = s2;
                    const long q = xs[0] + (long)nx * (xs[1] + (long)ny * xs[2]);
                    real fq[Q];
                    for (int i = 0; i < Q; ++i) fq[i] = c->f[FI(i, q)];
                    hecht_harting_cell(fq, a, face, face ? c->u_hi[a] : c->u_lo[a]);
                    for (int i = 0; i < Q; ++i) c->f[FI(i, q)] = fq[i];
                }
        }
    }
}

/* O-3: collide every cell, then stream: periodic axes wrap (L217); a link leaving through a wall
 * face is bounced back into the opposite direction at the same cell with Ladd's moving-wall
 * term, f_new,ibar(x) = f*_i(x) - 6 w_i rho_w (c_i.u_w), rho_w = 1 (G9: halfway bounce-back,
 * walls half a spacing outside the first/last fluid layer).  Corner rule: the wall velocity is
 * that of the first wall axis (x, y, z order) the link leaves through. */
int orc_step(orc_ctx* c, const double* g) {
    if (!c) return -1;
    const long N = c->cells;
    const int nx = c->n[0], ny = c->n[1], nz = c->n[2];
#pragma omp parallel for schedule(static)
    for (long q = 0; q < N; ++q) {
        real fin[Q], fout[Q], gq[3];
        for (int i = 0; i < Q; ++i) fin[i] = c->f[FI(i, q)];
        for (int d = 0; d < 3; ++d) gq[d] = g ? (real)g[(size_t)d * N + q] : 0;
        collide_cell(c, fin, gq, fout);
        for (int i = 0; i < Q; ++i) c->fstar[FI(i, q)] = fout[i];
        for (int d = 0; d < 3; ++d) c->g_last[(size_t)d * N + q] = gq[d];
    }
#pragma omp parallel for schedule(static)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                const long q = x + (long)nx * (y + (long)ny * z);
                const int xs[3] = {x, y, z};
                for (int i = 0; i < Q; ++i) {
                    int xp[3], leaves = 0;
                    const real* uw = NULL;
                    for (int a = 0; a < 3; ++a) {
                        xp[a] = xs[a] + C[i][a];
                        if (xp[a] < 0) {
                            if (c->kind[a] == ORC_PERIODIC) xp[a] += c->n[a];
                            else if (c->kind[a] == ORC_WALL_HH) leaves = 1;
                            else if (!uw) uw = c->u_lo[a];
                        } else if (xp[a] >= c->n[a]) {
                            if (c->kind[a] == ORC_PERIODIC) xp[a] -= c->n[a];
                            else if (c->kind[a] == ORC_WALL_HH) leaves = 1;
                            else if (!uw) uw = c->u_hi[a];
                        }
                    }
                    const real fs = c->fstar[FI(i, q)];
                    if (leaves) continue;      /* on-site wall: the population leaves the domain */
                    if (uw) {
                        real cu = C[i][0] * uw[0] + C[i][1] * uw[1] + C[i][2] * uw[2];
                        c->f[FI(OPP[i], q)] = fs - (real)6 * (real)weight(i) * (real)1 * cu;
                    } else {
                        const long qp = xp[0] + (long)nx * (xp[1] + (long)ny * xp[2]);
                        c->f[FI(i, qp)] = fs;
                    }
                }
            }
    hecht_harting_faces(c);
    return 0;
}

/* O-4: rho = sum f_i (Eq. 17); v = (sum c_i f_i + g_last/2)/rho (Eq. 18) */
int orc_read_macros(orc_ctx* c, double* rho, double* u) {
    if (!c) return -1;
    const long N = c->cells;
#pragma omp parallel for schedule(static)
    for (long q = 0; q < N; ++q) {
        real r = 0, j[3] = {0, 0, 0};
        for (int i = 0; i < Q; ++i) {
            real fi = c->f[FI(i, q)];
            r += fi;
            for (int d = 0; d < 3; ++d) j[d] += C[i][d] * fi;
        }
        if (rho) rho[q] = (double)r;
        if (u)
            for (int d = 0; d < 3; ++d) u[(size_t)d * N + q] = (double)((j[d] + c->g_last[(size_t)d * N + q] / 2) / r);
    }
    return 0;
}

int orc_read_populations(orc_ctx* c, double* f) {
    if (!c || !f) return -1;
#pragma omp parallel for schedule(static)
    for (long q = 0; q < c->cells; ++q)
        for (int i = 0; i < Q; ++i) f[(size_t)i * c->cells + q] = (double)c->f[FI(i, q)];
    return 0;
}
int orc_write_populations(orc_ctx* c, const double* f) {
    if (!c || !f) return -1;
#pragma omp parallel for schedule(static)
    for (long q = 0; q < c->cells; ++q)
        for (int i = 0; i < Q; ++i) c->f[FI(i, q)] = (real)f[(size_t)i * c->cells + q];
    hecht_harting_faces(c);
    return 0;
}

/* ------------------------------------------------------------------------------------------ */
int orc_add_mesh(orc_ctx* c, int n_nodes, const double* xyz, int n_edges, const int* edges,
                 const double* rest, double k, int* out_mesh_id) {
    if (!c || n_nodes < 1 || !xyz || n_edges < 0 || (n_edges && !edges)) return -1;
    for (int e = 0; e < n_edges; ++e)
        if (edges[2 * e] < 0 || edges[2 * e] >= n_nodes || edges[2 * e + 1] < 0 || edges[2 * e + 1] >= n_nodes ||
            edges[2 * e] == edges[2 * e + 1])
            return -1;
    if (c->n_nodes + n_nodes > c->cap_nodes) {
        c->cap_nodes = 2 * (c->n_nodes + n_nodes);
        c->X = (real*)realloc(c->X, (size_t)3 * c->cap_nodes * sizeof(real));
        c->F = (real*)realloc(c->F, (size_t)3 * c->cap_nodes * sizeof(real));
        c->U = (real*)realloc(c->U, (size_t)3 * c->cap_nodes * sizeof(real));
    }
    if (c->n_edges + n_edges > c->cap_edges) {
        c->cap_edges = 2 * (c->n_edges + n_edges);
        c->edge = (int*)realloc(c->edge, (size_t)2 * c->cap_edges * sizeof(int));
        c->rest = (real*)realloc(c->rest, (size_t)c->cap_edges * sizeof(real));
        c->kspring = (real*)realloc(c->kspring, (size_t)c->cap_edges * sizeof(real));
    }
    const int off = c->n_nodes;
    for (int m = 0; m < 3 * n_nodes; ++m) {
        c->X[3 * off + m] = (real)xyz[m];
        c->F[3 * off + m] = 0;
        c->U[3 * off + m] = 0;
    }
    for (int e = 0; e < n_edges; ++e) {
        const int a = edges[2 * e], b = edges[2 * e + 1], ge = c->n_edges + e;
        c->edge[2 * ge] = off + a;
        c->edge[2 * ge + 1] = off + b;
        if (rest) c->rest[ge] = (real)rest[e];
        else {
            double s = 0;
            for (int d = 0; d < 3; ++d) s += (xyz[3 * b + d] - xyz[3 * a + d]) * (xyz[3 * b + d] - xyz[3 * a + d]);
            c->rest[ge] = (real)sqrt(s);
        }
        c->kspring[ge] = (real)k;
    }
    c->n_nodes += n_nodes;
    c->n_edges += n_edges;
    if (out_mesh_id) *out_mesh_id = c->n_meshes;
    c->n_meshes += 1;
    c->mesh_off = (int*)realloc(c->mesh_off, (size_t)(c->n_meshes + 1) * sizeof(int));
    c->mesh_off[c->n_meshes - 1] = off;
    c->mesh_off[c->n_meshes] = c->n_nodes;
    c->mesh_edge_off = (int*)realloc(c->mesh_edge_off, (size_t)(c->n_meshes + 1) * sizeof(int));
    c->mesh_edge_off[c->n_meshes - 1] = c->n_edges - n_edges;
    c->mesh_edge_off[c->n_meshes] = c->n_edges;
    c->S0_tot = (real*)realloc(c->S0_tot, (size_t)c->n_meshes * sizeof(real));
    c->V0 = (real*)realloc(c->V0, (size_t)c->n_meshes * sizeof(real));
    c->k_s = (real*)realloc(c->k_s, (size_t)c->n_meshes * sizeof(real));
    c->k_t = (real*)realloc(c->k_t, (size_t)c->n_meshes * sizeof(real));
    c->k_v = (real*)realloc(c->k_v, (size_t)c->n_meshes * sizeof(real));
    c->S0_tot[c->n_meshes - 1] = c->V0[c->n_meshes - 1] = 0;
    c->k_s[c->n_meshes - 1] = c->k_t[c->n_meshes - 1] = c->k_v[c->n_meshes - 1] = 0;
    c->forces_valid = 0;
    return 0;
}

/* ---- NEXT-2: area and volume constraints (Eq. 4-5) -------------------------------
 *   H_area   = k_s (S_tot - S0_tot)^2 / (2 S0_tot) + sum_triangles k_t (S - S_0)^2 / (2 S_0)
 *   H_volume = k_v (V - V_0)^2 / (2 V_0)
 * with, for a triangle (a, b, c) oriented outwards,  n = (X_b - X_a) x (X_c - X_a),  S = |n|/2,
 * and for the closed surface  V = (1/6) sum_triangles X_a . (X_b x X_c)  (divergence theorem).
 * Nodal force = -dH/dX (Eq. 11 read with the minus sign, G2):
 *   dS/dX_a = (1/2) nhat x (X_c - X_b)   (cyclic in a, b, c),     dV/dX_a = (1/6) X_b x X_c  (cyclic). */
static void cross3(const real a[3], const real b[3], real out[3]) {
    out[0] = a[1] * b[2] - a[2] * b[1];
    out[1] = a[2] * b[0] - a[0] * b[2];
    out[2] = a[0] * b[1] - a[1] * b[0];
}
static real tri_area(const real* X, const int t[3], real nhat[3]) {
    real ab[3], ac[3], n[3];
    for (int d = 0; d < 3; ++d) {
        ab[d] = X[3 * t[1] + d] - X[3 * t[0] + d];
        ac[d] = X[3 * t[2] + d] - X[3 * t[0] + d];
    }
    cross3(ab, ac, n);
    const real len = (real)sqrt((double)(n[0] * n[0] + n[1] * n[1] + n[2] * n[2]));
    if (nhat)
        for (int d = 0; d < 3; ++d) nhat[d] = len > 0 ? n[d] / len : 0;
    return len / 2;
}
static real tri_volume6(const real* X, const int t[3]) {   /* X_a . (X_b x X_c) */
    real bc[3];
    cross3(X + 3 * t[1], X + 3 * t[2], bc);
    return X[3 * t[0]] * bc[0] + X[3 * t[0] + 1] * bc[1] + X[3 * t[0] + 2] * bc[2];
}
/* S_tot and V of mesh s at positions X */
static void mesh_area_volume(const orc_ctx* c, const real* X, int s, real* S_tot, real* V) {
    real S = 0, V6 = 0;
    for (int t = 0; t < c->n_tris; ++t) {
        if (c->tri_mesh[t] != s) continue;
        S += tri_area(X, c->tri + 3 * t, NULL);
        V6 += tri_volume6(X, c->tri + 3 * t);
    }
    *S_tot = S;
    *V = V6 / 6;
}

int orc_set_triangles(orc_ctx* c, int mesh_id, int n_tris, const int* tris, const double* ref_xyz,
                      double k_s, double k_t, double k_v) {
    if (!c || mesh_id < 0 || mesh_id >= c->n_meshes || n_tris < 1 || !tris) return -1;
    if (c->S0_tot[mesh_id] != 0) return -4;                       /* once per mesh */
    const int off = c->mesh_off[mesh_id], nn = c->mesh_off[mesh_id + 1] - off;
    for (int t = 0; t < 3 * n_tris; ++t)
        if (tris[t] < 0 || tris[t] >= nn) return -1;
    if (c->n_tris + n_tris > c->cap_tris) {
        c->cap_tris = 2 * (c->n_tris + n_tris);
        c->tri = (int*)realloc(c->tri, (size_t)3 * c->cap_tris * sizeof(int));
        c->tri_mesh = (int*)realloc(c->tri_mesh, (size_t)c->cap_tris * sizeof(int));
        c->tri_S0 = (real*)realloc(c->tri_S0, (size_t)c->cap_tris * sizeof(real));
    }
    /* the unstressed shape: ref_xyz (mesh-local node order), or the current positions */
    real* R = (real*)malloc((size_t)3 * c->n_nodes * sizeof(real));
    for (int m = 0; m < 3 * c->n_nodes; ++m) R[m] = c->X[m];
    if (ref_xyz)
        for (int m = 0; m < 3 * nn; ++m) R[3 * off + m] = (real)ref_xyz[m];
    for (int t = 0; t < n_tris; ++t) {
        const int gt = c->n_tris + t;
        for (int v = 0; v < 3; ++v) c->tri[3 * gt + v] = off + tris[3 * t + v];
        c->tri_mesh[gt] = mesh_id;
        c->tri_S0[gt] = tri_area(R, c->tri + 3 * gt, NULL);
        if (!(c->tri_S0[gt] > 0)) { free(R); return -1; }
    }
    c->n_tris += n_tris;
    mesh_area_volume(c, R, mesh_id, &c->S0_tot[mesh_id], &c->V0[mesh_id]);
    free(R);
    if (!(c->V0[mesh_id] > 0)) return -1;                         /* not closed / not outward oriented */
    c->k_s[mesh_id] = (real)k_s; c->k_t[mesh_id] = (real)k_t; c->k_v[mesh_id] = (real)k_v;
    c->forces_valid = 0;
    return 0;
}

int orc_mesh_area_volume(orc_ctx* c, int mesh_id, double* S_tot, double* V) {
    if (!c || mesh_id < 0 || mesh_id >= c->n_meshes) return -1;
    real S, Vv;
    mesh_area_volume(c, c->X, mesh_id, &S, &Vv);
    if (S_tot) *S_tot = (double)S;
    if (V) *V = (double)Vv;
    return 0;
}

/* H_area + H_volume of all meshes (Eq. 4-5) at the current positions */
double orc_area_volume_energy(orc_ctx* c) {
    double H = 0;
    for (int s = 0; s < c->n_meshes; ++s) {
        if (c->S0_tot[s] == 0) continue;
        real S, V;
        mesh_area_volume(c, c->X, s, &S, &V);
        H += 0.5 * (double)c->k_s[s] * (double)(S - c->S0_tot[s]) * (double)(S - c->S0_tot[s]) / (double)c->S0_tot[s];
        H += 0.5 * (double)c->k_v[s] * (double)(V - c->V0[s]) * (double)(V - c->V0[s]) / (double)c->V0[s];
    }
    for (int t = 0; t < c->n_tris; ++t) {
        const double S = (double)tri_area(c->X, c->tri + 3 * t, NULL), S0 = (double)c->tri_S0[t];
        H += 0.5 * (double)c->k_t[c->tri_mesh[t]] * (S - S0) * (S - S0) / S0;
    }
    return H;
}

/* F_m -= dH_area/dX_m + dH_volume/dX_m, triangle by triangle */
static void area_volume_forces(orc_ctx* c) {
    if (c->n_tris == 0) return;
    real* alpha = (real*)malloc((size_t)c->n_meshes * sizeof(real));   /* k_s (S_tot - S0_tot)/S0_tot */
    real* beta = (real*)malloc((size_t)c->n_meshes * sizeof(real));    /* k_v (V - V_0)/V_0 */
    for (int s = 0; s < c->n_meshes; ++s) {
        alpha[s] = beta[s] = 0;
        if (c->S0_tot[s] == 0) continue;
        real S, V;
        mesh_area_volume(c, c->X, s, &S, &V);
        alpha[s] = c->k_s[s] * (S - c->S0_tot[s]) / c->S0_tot[s];
        beta[s] = c->k_v[s] * (V - c->V0[s]) / c->V0[s];
    }
    for (int t = 0; t < c->n_tris; ++t) {
        const int* tv = c->tri + 3 * t;
        const int s = c->tri_mesh[t];
        real nhat[3];
        const real S = tri_area(c->X, tv, nhat);
        const real coefS = alpha[s] + c->k_t[s] * (S - c->tri_S0[t]) / c->tri_S0[t];
        for (int v = 0; v < 3; ++v) {
            const int a = tv[v], b = tv[(v + 1) % 3], cc = tv[(v + 2) % 3];
            real cb[3], dS[3], dV[3];
            for (int d = 0; d < 3; ++d) cb[d] = c->X[3 * cc + d] - c->X[3 * b + d];
            cross3(nhat, cb, dS);                               /* 2 dS/dX_a */
            cross3(c->X + 3 * b, c->X + 3 * cc, dV);            /* 6 dV/dX_a */
            for (int d = 0; d < 3; ++d) c->F[3 * a + d] -= coefS * dS[d] / 2 + beta[s] * dV[d] / 6;
        }
    }
    free(alpha); free(beta);
}

static int adhesion_forces(orc_ctx* c);   /* NEXT-4, below */

/* O-5: F <- 0; for each edge (a,b): R = X_b - X_a, l = |R|, e = k (l - L) R / l; F_a += e,
 * F_b -= e.  Eq. 2-3 (L92-99) with the sign read per G1: the force on point i is -grad_{X_i} of
 * Eq. 2, i.e. +k(|R|-L)R/|R| with R = X_j - X_i (attracting when stretched).  If sigma > 0,
 * F_m,d += sigma z_d(m, step): Philox normals keyed on (global node m, step, tag 2). */
int orc_compute_membrane_forces(orc_ctx* c, double sigma, uint64_t seed, uint64_t step) {
    if (!c) return -1;
    for (int m = 0; m < 3 * c->n_nodes; ++m) c->F[m] = 0;
    /* the edges of a mesh touch only that mesh's nodes: meshes are independent, and inside a mesh
     * the edges are visited in their given order */
    int zero_edge = 0;
#pragma omp parallel for schedule(dynamic, 1) reduction(| : zero_edge)
    for (int s = 0; s < c->n_meshes; ++s)
        for (int e = c->mesh_edge_off[s]; e < c->mesh_edge_off[s + 1]; ++e) {
            const int a = c->edge[2 * e], b = c->edge[2 * e + 1];
            real R[3], l2 = 0;
            for (int d = 0; d < 3; ++d) {
                R[d] = c->X[3 * b + d] - c->X[3 * a + d];
                l2 += R[d] * R[d];
            }
            const real l = (real)sqrt((double)l2);
            if (!(l > 0)) {
                zero_edge = 1;
                continue;
            }
            for (int d = 0; d < 3; ++d) {
                const real ed = c->kspring[e] * (l - c->rest[e]) * R[d] / l;
                c->F[3 * a + d] += ed;
                c->F[3 * b + d] -= ed;
            }
        }
    if (zero_edge) return -1;
    area_volume_forces(c);
    int rc = adhesion_forces(c);
    if (rc) return rc;
    if (sigma > 0)
#pragma omp parallel for schedule(static)
        for (int m = 0; m < c->n_nodes; ++m) {
            double z[3];
            orc_noise_normal3(seed, (uint64_t)m, (uint32_t)step, 2u, z);
            for (int d = 0; d < 3; ++d) c->F[3 * m + d] += (real)(sigma * z[d]);
        }
    c->forces_valid = 1;
    return 0;
}

double orc_spring_energy(orc_ctx* c) {
    double H = 0;
    for (int e = 0; e < c->n_edges; ++e) {
        const int a = c->edge[2 * e], b = c->edge[2 * e + 1];
        double l2 = 0;
        for (int d = 0; d < 3; ++d) {
            double r = (double)c->X[3 * b + d] - (double)c->X[3 * a + d];
            l2 += r * r;
        }
        const double dl = sqrt(l2) - (double)c->rest[e];
        H += 0.5 * (double)c->kspring[e] * dl * dl;     /* Eq. 2 (L94) */
    }
    return H;
}

/* Stencil of node X (O-6/O-7): base b_d = floor(X_d) - 1; cells q_d = b_d + o_d, o in {0..3}^3;
 * weight W = prod_d phi(X_d - q_d) (Eq. 35-36 with h = 1, so h^3 delta_h = phi phi phi);
 * periodic axes: index q_d mod n_d; wall axes: the cell is skipped if outside (G15).
 * Returns the wrapped linear cell index or -1 if dropped. */
static long stencil_cell(const orc_ctx* c, const real X[3], const int o[3], real* W) {
    long idx[3];
    real w = 1;
    for (int d = 0; d < 3; ++d) {
        const long b = (long)floor((double)X[d]) - 1;
        long qd = b + o[d];
        w *= phi(X[d] - (real)qd);
        if (c->kind[d] == ORC_PERIODIC) {
            qd %= c->n[d];
            if (qd < 0) qd += c->n[d];
        } else if (qd < 0 || qd >= c->n[d]) {
            *W = 0;
            return -1;
        }
        idx[d] = qd;
    }
    *W = w;
    return idx[0] + (long)c->n[0] * (idx[1] + (long)c->n[1] * idx[2]);
}

/* O-6: g_ijk = sum_m F_m phi phi phi (Eq. 34); g starts from zero each step. */
int orc_spread(orc_ctx* c, double* g) {
    if (!c || !g) return -1;
    if (c->n_nodes && !c->forces_valid) return -4;
    const long N = c->cells;
    real* acc = (real*)malloc((size_t)3 * N * sizeof(real));
#pragma omp parallel for schedule(static)
    for (long s = 0; s < 3 * N; ++s) acc[s] = 0;
    /* mesh by mesh; the stencils of different meshes may share cells, hence the atomic add */
#pragma omp parallel for schedule(dynamic, 1)
    for (int s = 0; s < c->n_meshes; ++s)
        for (int m = c->mesh_off[s]; m < c->mesh_off[s + 1]; ++m)
            for (int oz = 0; oz < 4; ++oz)
                for (int oy = 0; oy < 4; ++oy)
                    for (int ox = 0; ox < 4; ++ox) {
                        const int o[3] = {ox, oy, oz};
                        real W;
                        const long q = stencil_cell(c, &c->X[3 * m], o, &W);
                        if (q < 0) continue;
                        for (int d = 0; d < 3; ++d) {
                            const real add = W * c->F[3 * m + d];
#pragma omp atomic
                            acc[(size_t)d * N + q] += add;
                        }
                    }
#pragma omp parallel for schedule(static)
    for (long s = 0; s < 3 * N; ++s) g[s] = (double)acc[s];
    free(acc);
    return 0;
}

static void interpolate(const orc_ctx* c, const real* w /*3*cells*/, real* U) {
    const long N = c->cells;
#pragma omp parallel for schedule(static)
    for (int m = 0; m < c->n_nodes; ++m) {
        real Um[3] = {0, 0, 0};
        for (int oz = 0; oz < 4; ++oz)
            for (int oy = 0; oy < 4; ++oy)
                for (int ox = 0; ox < 4; ++ox) {
                    const int o[3] = {ox, oy, oz};
                    real W;
                    const long q = stencil_cell(c, &c->X[3 * m], o, &W);
                    if (q < 0) continue;
                    for (int d = 0; d < 3; ++d) Um[d] += W * w[(size_t)d * N + q];
                }
        for (int d = 0; d < 3; ++d) U[3 * m + d] = Um[d];
    }
}

int orc_interpolate_field(orc_ctx* c, const double* w, double* U) {
    if (!c || !w || !U) return -1;
    const long N = c->cells;
    real* wr = (real*)malloc((size_t)3 * N * sizeof(real));
    real* Ur = (real*)malloc((size_t)3 * (c->n_nodes + 1) * sizeof(real));
    for (size_t s = 0; s < (size_t)3 * N; ++s) wr[s] = (real)w[s];
    interpolate(c, wr, Ur);
    for (int m = 0; m < 3 * c->n_nodes; ++m) U[m] = (double)Ur[m];
    free(wr); free(Ur);
    return 0;
}

/* O-7: U_m = sum_ijk v_ijk phi phi phi (Eq. 33) with v the macroscopic velocity of the
 * CURRENT lattice state (after orc_step; reading A of G11: v = (sum c f^{n+1} + g^n/2)/rho^{n+1})
 * and the stencil around the not-yet-moved X_m (G13); then X_m <- X_m + U_m (forward Euler, G12;
 * Fig. 1 "positions were updated based on the velocities").  Positions stay unwrapped (G17).
 * Returns -5 if a node left the channel through a wall axis (X_d outside [-1/2, n_d - 1/2]). */
int orc_interpolate_advance(orc_ctx* c) {
    if (!c) return -1;
    const long N = c->cells;
    real* v = (real*)malloc((size_t)3 * N * sizeof(real));
#pragma omp parallel for schedule(static)
    for (long q = 0; q < N; ++q) {
        real r = 0, j[3] = {0, 0, 0};
        for (int i = 0; i < Q; ++i) {
            real fi = c->f[FI(i, q)];
            r += fi;
            for (int d = 0; d < 3; ++d) j[d] += C[i][d] * fi;
        }
        for (int d = 0; d < 3; ++d) v[(size_t)d * N + q] = (j[d] + c->g_last[(size_t)d * N + q] / 2) / r;
    }
    interpolate(c, v, c->U);
    free(v);
    int left = 0;
#pragma omp parallel for schedule(static) reduction(| : left)
    for (int m = 0; m < c->n_nodes; ++m)
        for (int d = 0; d < 3; ++d) {
            c->X[3 * m + d] += c->U[3 * m + d];
            if (c->kind[d] == ORC_WALL &&
                (c->X[3 * m + d] < (real)-0.5 || c->X[3 * m + d] > (real)c->n[d] - (real)0.5))
                left = 1;
            if (c->kind[d] == ORC_WALL_HH &&        /* on-site walls lie ON layers 0 and n - 1 */
                (c->X[3 * m + d] < (real)0 || c->X[3 * m + d] > (real)c->n[d] - (real)1))
                left = 1;
        }
    c->forces_valid = 0;
    return left ? -5 : 0;
}

int orc_n_nodes(orc_ctx* c) { return c ? c->n_nodes : -1; }
int orc_read_nodes(orc_ctx* c, double* xyz) {
    if (!c || !xyz) return -1;
    for (int m = 0; m < 3 * c->n_nodes; ++m) xyz[m] = (double)c->X[m];
    return 0;
}
int orc_write_nodes(orc_ctx* c, const double* xyz) {
    if (!c || !xyz) return -1;
    for (int m = 0; m < 3 * c->n_nodes; ++m) c->X[m] = (real)xyz[m];
    c->forces_valid = 0;
    return 0;
}
int orc_read_forces(orc_ctx* c, double* F) {
    if (!c || !F) return -1;
    for (int m = 0; m < 3 * c->n_nodes; ++m) F[m] = (double)c->F[m];
    return 0;
}
int orc_write_forces(orc_ctx* c, const double* F) {
    if (!c || !F) return -1;
    for (int m = 0; m < 3 * c->n_nodes; ++m) c->F[m] = (real)F[m];
    c->forces_valid = 1;
    return 0;
}
int orc_read_node_velocities(orc_ctx* c, double* U) {
    if (!c || !U) return -1;
    for (int m = 0; m < 3 * c->n_nodes; ++m) U[m] = (double)c->U[m];
    return 0;
}

/* =============================================================================================
 * NEXT-4: stochastic dynamic adhesion model (section 3.2) + wall repulsion (section 3.4.1).
 * Decision arithmetic (probabilities, capture distance) is fp64 in BOTH builds and on the GPU:
 * a Monte-Carlo decision is an integer outcome, so both sides take it in the same precision.
 * ============================================================================================= */
static void tangential_axes(int a, int* t0, int* t1) {
    *t0 = a == 0 ? 1 : 0;
    *t1 = a == 2 ? 1 : 2;
}
static double wall_plane(const orc_ctx* c, int a) { return c->kind[a] == ORC_WALL_HH ? 0.0 : -0.5; }

int orc_set_receptors(orc_ctx* c, int n_rec, const int* node, const orc_adhesion* prm) {
    if (!c || n_rec < 0 || (n_rec && !node) || !prm) return -1;
    const int a = prm->wall_axis;
    if (a < 0 || a > 2 || c->kind[a] == ORC_PERIODIC || prm->max_per_site < 1) return -1;
    if (!(prm->l_max > 0) || prm->k_on0 < 0 || prm->k_off0 < 0) return -1;
    for (int r = 0; r < n_rec; ++r)
        if (node[r] < 0 || node[r] >= c->n_nodes) return -1;
    int t0, t1;
    tangential_axes(a, &t0, &t1);
    free(c->rec_node); free(c->bond); free(c->site_count);
    c->n_rec = n_rec;
    c->rec_node = (int*)malloc(sizeof(int) * (size_t)(n_rec > 0 ? n_rec : 1));
    c->bond = (int*)calloc((size_t)3 * (size_t)(n_rec > 0 ? n_rec : 1), sizeof(int));
    c->site_count = (int*)calloc((size_t)c->n[t0] * (size_t)c->n[t1], sizeof(int));
    for (int r = 0; r < n_rec; ++r) c->rec_node[r] = node[r];
    c->adh = *prm;
    c->forces_valid = 0;
    return 0;
}

/* linear index of site (s0, s1) for the per-site bond count, -1 if the site does not exist
 * (outside a non-periodic tangential axis) */
static long site_index(const orc_ctx* c, int t0, int t1, long s0, long s1) {
    long s[2] = {s0, s1};
    const int t[2] = {t0, t1};
    for (int e = 0; e < 2; ++e) {
        const long n = c->n[t[e]];
        if (c->kind[t[e]] == ORC_PERIODIC) {
            s[e] %= n;
            if (s[e] < 0) s[e] += n;
        } else if (s[e] < 0 || s[e] >= n) {
            return -1;
        }
    }
    return s[0] + (long)c->n[t0] * s[1];
}

/* distance between the receptor at X and the site (s0, s1) on the wall plane */
static double bond_length(const orc_ctx* c, const real* X, int a, int t0, int t1, long s0, long s1, double R[3]) {
    R[a] = wall_plane(c, a) - (double)X[a];
    R[t0] = (double)s0 - (double)X[t0];
    R[t1] = (double)s1 - (double)X[t1];
    return sqrt(R[0] * R[0] + R[1] * R[1] + R[2] * R[2]);
}

void orc_adhesion_probabilities(const orc_adhesion* p, double x_b, double* P_f, double* P_r) {
    const double d = fabs(x_b - p->l_b);
    const double k_on = p->k_on0 * exp(p->s * d * (p->gamma - 0.5 * d));   /* Eq. 13 */
    const double k_off = p->k_off0 * exp(p->gamma * p->s * d);             /* Eq. 12, F_b = sigma d */
    if (P_f) *P_f = 1.0 - exp(-k_on);                                      /* L151, dt = 1 */
    if (P_r) *P_r = 1.0 - exp(-k_off);
}

int orc_adhesion_update(orc_ctx* c, uint64_t seed, uint64_t step) {
    if (!c || !c->rec_node) return -4;
    const orc_adhesion* p = &c->adh;
    const int a = p->wall_axis;
    int t0, t1;
    tangential_axes(a, &t0, &t1);
    /* 1) break the already formed bonds (L276) */
    for (int r = 0; r < c->n_rec; ++r) {
        int* b = c->bond + 3 * r;
        if (!b[0]) continue;
        double R[3], xi[4], P_r;
        const double x_b = bond_length(c, c->X + 3 * c->rec_node[r], a, t0, t1, b[1], b[2], R);
        orc_adhesion_probabilities(p, x_b, NULL, &P_r);
        orc_noise_uniform(seed, (uint64_t)r, (uint32_t)step, 3u, xi);
        if (xi[0] < P_r) {
            c->site_count[site_index(c, t0, t1, b[1], b[2])] -= 1;
            b[0] = 0; b[1] = 0; b[2] = 0;                            /* an open receptor names no site */
        }
    }
    /* 2) generate new bonds from unbound receptors and sites with a free place (L147-149, L276):
     * receptor order = index order, so the lowest indices take the free places of a site */
    for (int r = 0; r < c->n_rec; ++r) {
        int* b = c->bond + 3 * r;
        if (b[0]) continue;                                          /* rule 1: one vWF per receptor */
        const real* X = c->X + 3 * c->rec_node[r];
        const long s0 = (long)floor((double)X[t0] + 0.5), s1 = (long)floor((double)X[t1] + 0.5);   /* nearest site */
        const long si = site_index(c, t0, t1, s0, s1);
        if (si < 0) continue;
        double R[3], xi[4], P_f;
        const double x_b = bond_length(c, X, a, t0, t1, s0, s1, R);
        if (!(x_b < p->l_max)) continue;                             /* L149: closer than the bond length */
        if (c->site_count[si] >= p->max_per_site) continue;          /* rule 2: at most 4 receptors per vWF */
        orc_adhesion_probabilities(p, x_b, &P_f, NULL);
        orc_noise_uniform(seed, (uint64_t)r, (uint32_t)step, 3u, xi);
        if (xi[1] < P_f) {
            b[0] = 1; b[1] = (int)s0; b[2] = (int)s1;
            c->site_count[si] += 1;
        }
    }
    c->forces_valid = 0;
    return 0;
}

int orc_read_bonds(orc_ctx* c, int* bonds) {
    if (!c || !bonds) return -1;
    for (int i = 0; i < 3 * c->n_rec; ++i) bonds[i] = c->bond[i];
    return 0;
}

int orc_write_bonds(orc_ctx* c, const int* bonds) {
    if (!c || !bonds || !c->rec_node) return -1;
    int t0, t1;
    tangential_axes(c->adh.wall_axis, &t0, &t1);
    const long n_sites = (long)c->n[t0] * c->n[t1];
    for (long i = 0; i < n_sites; ++i) c->site_count[i] = 0;
    for (int r = 0; r < c->n_rec; ++r) {
        int* b = c->bond + 3 * r;
        b[0] = bonds[3 * r] ? 1 : 0; b[1] = b[0] ? bonds[3 * r + 1] : 0; b[2] = b[0] ? bonds[3 * r + 2] : 0;
        if (b[0]) {
            const long si = site_index(c, t0, t1, b[1], b[2]);
            if (si < 0) return -1;
            c->site_count[si] += 1;
        }
    }
    c->forces_valid = 0;
    return 0;
}

/* Eq. 14 read as the restoring spring force of the bond on its node (magnitude sigma |x_b - l_b|,
 * towards the site when stretched), plus F_rep of L246 on every node along the inward normal. */
static int adhesion_forces(orc_ctx* c) {
    if (!c->rec_node) return 0;
    const orc_adhesion* p = &c->adh;
    const int a = p->wall_axis;
    int t0, t1;
    tangential_axes(a, &t0, &t1);
    for (int r = 0; r < c->n_rec; ++r) {
        const int* b = c->bond + 3 * r;
        if (!b[0]) continue;
        const int m = c->rec_node[r];
        double R[3];
        const double x_b = bond_length(c, c->X + 3 * m, a, t0, t1, b[1], b[2], R);
        if (!(x_b > 0)) continue;
        for (int d = 0; d < 3; ++d) c->F[3 * m + d] += (real)(p->sigma * (x_b - p->l_b) * R[d] / x_b);
    }
    if (p->F0 > 0)
        for (int m = 0; m < c->n_nodes; ++m) {
            const double eps = (double)c->X[3 * m + a] - wall_plane(c, a);
            if (!(eps > 0)) return -5;
            const double e = exp(-p->tau_rep * eps);
            c->F[3 * m + a] += (real)(p->F0 * p->tau_rep * e / (1.0 - e));
        }
    return 0;
}

double orc_adhesion_energy(orc_ctx* c) {
    if (!c || !c->rec_node) return 0.0;
    const orc_adhesion* p = &c->adh;
    const int a = p->wall_axis;
    int t0, t1;
    tangential_axes(a, &t0, &t1);
    double H = 0;
    for (int r = 0; r < c->n_rec; ++r) {
        const int* b = c->bond + 3 * r;
        if (!b[0]) continue;
        double R[3];
        const double x_b = bond_length(c, c->X + 3 * c->rec_node[r], a, t0, t1, b[1], b[2], R);
        H += 0.5 * p->sigma * (x_b - p->l_b) * (x_b - p->l_b);
    }
    if (p->F0 > 0)
        for (int m = 0; m < c->n_nodes; ++m) {
            const double eps = (double)c->X[3 * m + a] - wall_plane(c, a);
            H -= p->F0 * log(1.0 - exp(-p->tau_rep * eps));
        }
    return H;
}
