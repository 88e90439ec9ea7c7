/* oracle/orc.h -- CPU ORACLE, TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, obviously-correct implementation of the per-time-step fluid-structure hot path of
 * arXiv:1312.2234 (section 3.3, 3.4.2, Eq. 2-3, 15-21, 31-36), written from the paper.
 * It shares no code with the CUDA library.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call it; the product path never does.
 *
 * All pointers are HOST pointers.  All floating point arrays at this interface are double,
 * whatever the internal precision (the default build is fp64; -DORC_REAL_FLOAT builds the fp32
 * diagnostic mode).  Linear cell index q = i + nx*(j + ny*k); fields are SoA: rho[cells],
 * u[3*cells] = (ux[cells], uy[cells], uz[cells]); populations f[19*cells] = f_i at [i*cells + q]
 * with i = (paper's 1-based index) - 1, the order fixed by PAPER.md Eq. 23-30 (see orc.c).
 *
 * Return codes: 0 ok, -1 invalid argument, -4 wrong call order, -5 a node left the channel.
 */
#ifndef ORC_H
#define ORC_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct orc_ctx orc_ctx;

/* ORC_WALL: halfway bounce-back + Ladd term (configs, G9).  ORC_WALL_HH: the paper's own wall, the
 * Hecht-Harting on-site velocity condition (Eq. 23-30): wall ON the first/last layer; the other two
 * axes must be periodic. */
enum { ORC_PERIODIC = 0, ORC_WALL = 1, ORC_WALL_HH = 2 };

/* lattice constants: c[19][3] and w[19] in the paper's order (Eq. 21, Eq. 23-30) */
void orc_lattice(int* c_out /*19*3*/, double* w_out /*19*/);
int  orc_real_bytes(void);   /* 8 (fp64 build) or 4 (fp32 build) */

/* PAPER.md Eq. 36: phi(r) = (1 + cos(pi r / 2))/4 for |r| < 2, else 0 */
double orc_phi(double r);
/* PAPER.md Eq. 20 (one population, paper index i0 = i-1) */
double orc_feq(int i0, double rho, const double v[3]);
/* Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11) and the derived uniform / normal variates */
void   orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
double orc_uniform01(uint32_t r);                                  /* ((r>>8)+0.5) 2^-24 */
void   orc_noise_uniform(uint64_t seed, uint64_t index, uint32_t step, uint32_t tag, double xi[4]);
void   orc_noise_normal3(uint64_t seed, uint64_t index, uint32_t step, uint32_t tag, double z[3]);
void   orc_noise_normal3_many(uint64_t seed, const uint64_t* index, long n, uint32_t step, uint32_t tag, double* z);

int orc_create(int nx, int ny, int nz, double tau, const int kind[3],
               const double u_lo[9] /*[axis][comp]*/, const double u_hi[9], orc_ctx** out);
int orc_destroy(orc_ctx*);

/* f_i = feq_i(rho, u) + amp (2 xi - 1); rho NULL = 1, u NULL = 0 */
int orc_set_equilibrium(orc_ctx*, const double* rho, const double* u, double noise_amp, uint64_t seed);
/* one collide + stream + boundary step with force density g[3*cells] (NULL = 0) */
int orc_step(orc_ctx*, const double* g);
/* rho = sum f_i, v = (sum c_i f_i + g_last/2)/rho of the current state */
int orc_read_macros(orc_ctx*, double* rho, double* u);
int orc_read_populations(orc_ctx*, double* f /*19*cells*/);
int orc_write_populations(orc_ctx*, const double* f);

int orc_add_mesh(orc_ctx*, int n_nodes, const double* xyz /*AoS*/, int n_edges, const int* edges,
                 const double* rest /*NULL = lengths of xyz*/, double k, int* out_mesh_id);
/* NEXT-2 (Eq. 4-5): triangles (mesh-local node triples, outward orientation) of mesh mesh_id, the
 * unstressed shape ref_xyz (n_nodes x 3, NULL = the current positions) that defines S_0, S0_tot, V_0,
 * and the coefficients k_s (global area), k_t (local area), k_v (volume).  Once per mesh. */
int orc_set_triangles(orc_ctx*, int mesh_id, int n_tris, const int* tris, const double* ref_xyz,
                      double k_s, double k_t, double k_v);
int orc_mesh_area_volume(orc_ctx*, int mesh_id, double* S_tot, double* V);
double orc_area_volume_energy(orc_ctx*);   /* H_area + H_volume, Eq. 4-5 */
/* springs (Eq. 2-3) + area / volume constraint forces (Eq. 4-5, meshes with triangles) + noise */
int orc_compute_membrane_forces(orc_ctx*, double sigma, uint64_t seed, uint64_t step);
int orc_spread(orc_ctx*, double* g /*3*cells, overwritten*/);
int orc_interpolate_advance(orc_ctx*);
int orc_n_nodes(orc_ctx*);
int orc_read_nodes(orc_ctx*, double* xyz /*AoS*/);
int orc_write_nodes(orc_ctx*, const double* xyz);
int orc_read_forces(orc_ctx*, double* F /*AoS*/);
int orc_write_forces(orc_ctx*, const double* F);
int orc_read_node_velocities(orc_ctx*, double* U /*AoS, of the last interpolate*/);
/* Eq. 2 summed over all edges of all meshes: H_SCE = sum k/2 (|R| - L)^2 */
double orc_spring_energy(orc_ctx*);
/* U_m = sum_cells w[q] phi phi phi around the CURRENT node positions, for any field w[3*cells];
 * no advance (used for the adjointness pin) */
int orc_interpolate_field(orc_ctx*, const double* w, double* U /*AoS*/);

/* ---- NEXT-4: stochastic dynamic adhesion model (section 3.2, Eq. 12-14, rules L147-149)
 * and short-range wall repulsion (section 3.4.1).  DESIGN.md readings A-1 .. A-9.
 * All quantities in lattice units (h = dt = 1); rates are per time step.
 *   receptors : receptor r sits on global node node[r] ("located at ith node", Eq. 14)
 *   vWF sites : on the LOW face of wall axis `wall_axis`, one per lattice point of that plane
 *               (25 per um^2 = one per h^2 at h = 0.2 um, L145/L173); the plane lies at -1/2
 *               (ORC_WALL) or 0 (ORC_WALL_HH); a site is named by its two tangential integer
 *               coordinates (s0, s1), the tangential axes in x, y, z order, kept unwrapped
 *   k_on  = k_on0  exp( s d (gamma - d/2) ),  d = |x_b - l_b|,  s = sigma/(k_B T)     (Eq. 13)
 *   k_off = k_off0 exp( gamma s d )             (Eq. 12 with F_b = sigma d)
 *   P_f = 1 - exp(-k_on), P_r = 1 - exp(-k_off) (L151)
 *   bond force on the node: sigma (x_b - l_b) (S - X)/x_b                         (Eq. 14)
 *   repulsion on every node: F0 tau exp(-tau eps)/(1 - exp(-tau eps)) along the inward wall normal,
 *               eps = distance of the node from the wall plane                    (L246)     */
typedef struct {
    int    wall_axis;
    int    max_per_site;       /* rule 2 (L148): 4 */
    double k_on0, k_off0;
    double s;                  /* sigma / k_B T */
    double gamma;              /* reactive compliance (a length) */
    double sigma;              /* bond spring constant */
    double l_b, l_max;         /* equilibrium bond length; capture distance (128 nm, L149) */
    double F0, tau_rep;        /* repulsion (0 = off) */
} orc_adhesion;
int orc_set_receptors(orc_ctx*, int n_receptors, const int* node, const orc_adhesion* prm);
/* one Monte-Carlo update at the current node positions: first every existing bond is tested for
 * breakage, then every unbound receptor for formation (order of L276); random numbers from
 * Philox keyed on (seed; receptor, step, tag 3): word 0 breaks, word 1 forms. */
int orc_adhesion_update(orc_ctx*, uint64_t seed, uint64_t step);
int orc_read_bonds(orc_ctx*, int* bonds /*3 per receptor: bound, s0, s1*/);
int orc_write_bonds(orc_ctx*, const int* bonds);
/* sum over bonds sigma/2 (x_b - l_b)^2  -  F0 sum over nodes ln(1 - exp(-tau eps)): the potential
 * whose negative gradient the adhesion + repulsion forces are (for the finite-difference pin) */
double orc_adhesion_energy(orc_ctx*);
/* P_f and P_r at bond length x_b (the closed forms above) */
void orc_adhesion_probabilities(const orc_adhesion* prm, double x_b, double* P_f, double* P_r);

#ifdef __cplusplus
}
#endif
#endif
