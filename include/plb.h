/* plb.h -- C-ABI of libplb: the per-time-step fluid-structure hot path of arXiv:1312.2234
 * (Wu, Xu, Kim, Alber) as hand-written CUDA for one B200 (sm_100a).
 *
 * One coupled step (Fig. 1) is four calls, in this order:
 *     ib_compute_membrane_forces -> ib_spread -> lbm_step(forcing) -> ib_interpolate_advance
 *
 * Conventions
 *   - Lattice units h = dt = 1, c_s^2 = 1/3.  Lattice node (i,j,k) is the integer
 *     point (i,j,k) (L268); linear cell index q = i + nx*(j + ny*k), x fastest.
 *   - D3Q19, populations numbered as in the paper (Eq. 21 / Eq. 23-30): index i-1 at this
 *     interface.  c = +x,-x,+y,-y,+z,-z, +x+y,+x-y,+x+z,+x-z, -x+y,-x-y,-x+z,-x-z, +y+z,+y-z,
 *     -y+z,-y-z, 0; weights 2/36 (x6), 1/36 (x12), 12/36.
 *   - "d_" arguments are DEVICE pointers owned by the caller; "h_" arguments are HOST pointers,
 *     copied during the call (the caller keeps them).  No torch types cross this boundary.
 *   - Scalar fields are float[cells]; vector fields handed to lbm_set_equilibrium /
 *     lbm_read_macros are SoA float[3*cells] = (x[cells], y[cells], z[cells]).
 *   - The FORCING field is AoS: float4 per cell = (g_x, g_y, g_z, 0), 16-byte aligned, so that
 *     the spread can use 128-bit vector atomics.
 *   - The library never allocates device memory: the caller passes one workspace of
 *     lbm_workspace_bytes() bytes (256-byte aligned) to lbm_create, which carves it.  (One call,
 *     lbm_check_finite_static, keeps its scratch in a 256 KiB device array inside the library.)
 *   - Calls that take only device pointers are asynchronous on the context's stream.  Calls that
 *     take host pointers synchronise that stream before returning.
 *   - Every call returns 0 on success or a negative code (below); plb_last_error() gives a
 *     thread-local message.  No exceptions, no aborts, no printing.  There is NO CPU fallback:
 *     with no CUDA device every compute call fails with PLB_ERR_CUDA.
 */
#ifndef PLB_H
#define PLB_H
#include <stddef.h>
#if defined(__GNUC__)
#define PLB_API __attribute__((visibility("default")))
#else
#define PLB_API
#endif
#ifdef __cplusplus
extern "C" {
#endif

typedef struct plb_ctx plb_ctx; /* opaque */

typedef struct { int nx, ny, nz; } plb_grid;

enum { PLB_PERIODIC = 0, PLB_WALL_BB = 1, PLB_WALL_HH = 2 }; /* per axis */

/* kind[a]: PLB_PERIODIC wraps populations across axis a.  PLB_WALL_BB closes both
 * faces of axis a with link-wise halfway bounce-back: all n_a layers are fluid, the walls lie half
 * a spacing outside (at -1/2 and n_a - 1/2), a link leaving through a face returns into the
 * opposite direction at the same node with Ladd's moving-wall term -6 w_i rho_w (c_i . u_w),
 * rho_w = 1 (reading G9).  u_lo[a] / u_hi[a] = wall velocity at the low / high face of
 * axis a.  A link leaving through two wall faces at once takes the velocity of the first such
 * axis in x, y, z order.
 * PLB_WALL_HH is the wall the paper itself uses (L217-238): the Hecht-Harting on-site velocity
 * condition.  The walls lie ON layers 0 and n_a - 1; after streaming, the populations of a wall
 * cell that point into the fluid are "undetermined" and are closed from the others by Eq. 23-30
 * (printed for the plane z = 0; other faces by renaming the axes), which sets
 * sum_i c_i f_i = rho u_wall with rho from the first line of L219; wall cells then collide like
 * any other.  lbm_set_equilibrium / lbm_write_populations close the wall layers too (DESIGN.md
 * G24, G25).  Only one axis may be PLB_WALL_HH, the other two must be periodic, n_a >= 2. */
typedef struct {
    int   kind[3];
    float u_lo[3][3];
    float u_hi[3][3];
} plb_boundary;

enum {
    PLB_OK            =  0,
    PLB_ERR_ARG       = -1, /* invalid argument */
    PLB_ERR_WORKSPACE = -2, /* workspace too small / capacity exceeded */
    PLB_ERR_CUDA      = -3, /* CUDA error (message in plb_last_error) */
    PLB_ERR_ORDER     = -4, /* wrong call order (e.g. ib_spread before forces) */
    PLB_ERR_NODE_LEFT = -5  /* a node left the channel through a wall axis */
};

PLB_API const char* plb_last_error(void);

/* Bytes of workspace lbm_create needs for this grid and mesh capacity (two fp32 lattices, the
 * activity-segment mask and list, the (v, rho) field of the listed segments, node arrays, the
 * per-topology spring tables, node ranges and their boxes, triangle arrays). */
PLB_API int lbm_workspace_bytes(const plb_grid* grid, long max_nodes, long max_edges, size_t* out_bytes);

/* Create a context.  tau > 1/2 is the BGK relaxation time (Eq. 16).  d_workspace must stay
 * valid until lbm_destroy.  cuda_stream is a cudaStream_t (NULL = the legacy default stream).
 * The populations are undefined until lbm_set_equilibrium or lbm_write_populations. */
PLB_API int lbm_create(const plb_grid* grid, float tau, const plb_boundary* bnd, void* d_workspace,
               size_t workspace_bytes, long max_nodes, long max_edges, void* cuda_stream,
               plb_ctx** out);
PLB_API int lbm_destroy(plb_ctx* ctx); /* frees host bookkeeping only */

/* f_i = f_i^eq(rho, u) (Eq. 20) + noise_amp (2 xi - 1).  d_rho NULL = 1, d_u NULL = 0.
 * xi = Philox4x32-10 uniform keyed on (seed; index = cell*19 + (i-1), step 0, tag 1), first
 * output word, xi = ((r >> 8) + 1/2) 2^-24 (O-8).  Resets the step counter and g_last. */
PLB_API int lbm_set_equilibrium(plb_ctx* ctx, const float* d_rho, const float* d_u, float noise_amp,
                        unsigned long long seed);

/* One fused collide + stream + boundary step (Eq. 16-21 with the Guo forcing of Eq. 19, periodic
 * wrap L217, bounce-back as above).  d_forcing: float4 per cell, or NULL = no force.  When
 * d_forcing is the buffer ib_spread last filled, only the cells that spread touched are read.
 * LIFETIME: the library keeps the pointer.  The buffer must stay allocated and unmodified until
 * the next lbm_step, lbm_set_equilibrium, lbm_write_populations or lbm_destroy, because
 * ib_interpolate_advance and lbm_read_macros read it (they add g/2 to the momentum, L201). */
PLB_API int lbm_step(plb_ctx* ctx, const float* d_forcing);

/* rho = sum f_i (Eq. 17), v = (sum c_i f_i + g_last/2)/rho (Eq. 18) of the current state.
 * Either output may be NULL. */
PLB_API int lbm_read_macros(plb_ctx* ctx, float* d_rho, float* d_u);

/* Add one mesh (nodes = actin vertices, edges = filaments).  h_xyz: n_nodes x 3
 * doubles (AoS, unwrapped lattice coordinates); h_edges: n_edges x 2 mesh-local node indices;
 * h_rest: n_edges rest lengths L_ij (NULL = the lengths of h_xyz); k: spring stiffness of Eq. 2.
 * Meshes are concatenated; global node index = running offset + local index.  (Inside the
 * library the nodes of a mesh are stored in a different, spatially coherent order; every call
 * that names a node -- ib_read/write_*, ib_set_triangles, ib_set_receptors, the noise key --
 * speaks the caller's indices.) */
PLB_API int ib_add_mesh(plb_ctx* ctx, int n_nodes, const double* h_xyz, int n_edges, const int* h_edges,
                const float* h_rest, float k, int* out_mesh_id);
/* n_meshes meshes of identical topology and rest lengths: h_xyz is n_meshes x n_nodes x 3. */
PLB_API int ib_add_meshes(plb_ctx* ctx, int n_meshes, int n_nodes, const double* h_xyz, int n_edges,
                  const int* h_edges, const float* h_rest, float k, int* out_first_mesh_id);

/* Area and volume constraints of the lipid bilayer (Eq. 4-5)
 * for meshes first_mesh_id .. first_mesh_id + n_meshes - 1, which must share one topology:
 *   H_area   = k_s (S_tot - S0_tot)^2/(2 S0_tot) + sum_triangles k_t (S - S_0)^2/(2 S_0)
 *   H_volume = k_v (V - V_0)^2/(2 V_0)
 * h_tris: n_tris x 3 mesh-local node indices, oriented outwards (V_0 must come out positive; the
 * surface must be closed).  h_ref_xyz: n_nodes x 3 doubles, the unstressed shape that defines
 * S_0, S0_tot and V_0 (any rigid placement), or NULL = each mesh's current positions.  Once per
 * mesh.  Capacity: 2 * max_nodes triangles (a closed genus-0 surface of N nodes has 2N - 4).
 * From then on ib_compute_membrane_forces adds -dH/dX of these meshes to the spring forces. */
PLB_API int ib_set_triangles(plb_ctx* ctx, int first_mesh_id, int n_meshes, int n_tris, const int* h_tris,
                     const double* h_ref_xyz, float k_s, float k_t, float k_v);

/* S1.  F <- 0; for every edge (a,b): R = X_b - X_a, e = k (|R| - L) R/|R|, F_a += e, F_b -= e
 * (Eq. 2-3, sign read as F = -grad H, G1).  If noise_sigma > 0 adds
 * noise_sigma * N(0,1) per node component from Philox keyed on (noise_seed; global node, step,
 * tag 2) with Box-Muller (O-8).  Meshes given triangles by ib_set_triangles also get
 * the area / volume constraint forces of Eq. 4-5. */
PLB_API int ib_compute_membrane_forces(plb_ctx* ctx, float noise_sigma, unsigned long long noise_seed,
                               unsigned long long step);

/* S2.  g_ijk = sum_m F_m phi(i - X_m) phi(j - Y_m) phi(k - Z_m) (Eq. 34-36) with the
 * 4-point cosine kernel phi(r) = (1 + cos(pi r/2))/4, |r| < 2, over the 4x4x4 cells
 * floor(X) - 1 .. floor(X) + 2; periodic axes wrap the index, cells beyond a wall axis are
 * dropped.  d_forcing (float4 per cell) must have been zero-filled once by the caller; each call
 * first clears what the previous call wrote.  LIFETIME: the library keeps the pointer and the
 * next ib_spread WRITES zeros into the previous call's buffer, whichever buffer it is given: a
 * buffer handed to ib_spread must stay allocated until the second next ib_spread,
 * ib_release_forcing or lbm_destroy. */
PLB_API int ib_spread(plb_ctx* ctx, float* d_forcing);

/* The three forms of the S2 kernel (all compute the sum of Eq. 34; they differ in how the
 * contributions of the nodes of one thread block meet in its shared-memory lattice tile):
 *   SCATTER   one shared-memory atomic per (node, cell, component);
 *   AGGREGATE warp-aggregated atomics: a warp groups its 32 consecutive nodes by base cell
 *             (match.any), sums each group in registers and issues one shared-memory atomic per
 *             (group, cell, component);
 *   GATHER    nodes counting-sorted by base cell, one thread per tile cell sums over the 4 x 4 x 4
 *             base cells around it: no atomics (the form of the paper's own
 *             fluid3d_force_distribute_kernel, L356-362).
 * AUTO (default) picks SCATTER or AGGREGATE from the sampling density of the tiles (DESIGN.md
 * section 5 has the measurements behind the choice).  ib_get_spread_mode returns the form
 * ib_spread would launch now.
 * Whatever the form, ib_spread also LISTS every cell inside some node's stencil (also where the
 * spread force is zero): right after it, ib_interpolate_advance for the same positions reads the
 * velocity of exactly those cells. */
enum { PLB_SPREAD_AUTO = 0, PLB_SPREAD_SCATTER = 1, PLB_SPREAD_AGGREGATE = 2, PLB_SPREAD_GATHER = 3 };
PLB_API int ib_set_spread_mode(plb_ctx* ctx, int mode);
PLB_API int ib_get_spread_mode(plb_ctx* ctx, int* out_mode_in_use);

/* Forget the forcing buffers the context still points to (the one ib_spread last filled, the one
 * lbm_step last read), clearing what ib_spread wrote first; the caller may free them afterwards.
 * ib_interpolate_advance / lbm_read_macros then see g = 0 until the next lbm_step. */
PLB_API int ib_release_forcing(plb_ctx* ctx);

/* S4 + S5.  U_m = sum_ijk v_ijk phi phi phi (Eq. 33) with v the velocity lbm_read_macros
 * would return now (state after lbm_step, force just applied) and the stencil around the not yet
 * moved X_m; then X_m <- X_m + U_m (forward Euler).  Positions are kept unwrapped in fp64.
 * Needs no preceding ib_spread: lbm_step(NULL) -> ib_interpolate_advance is passive advection.
 * A node ending outside [-1/2, n_a - 1/2] on a wall axis raises a sticky flag that plb_status and
 * ib_read_nodes report as PLB_ERR_NODE_LEFT. */
PLB_API int ib_interpolate_advance(plb_ctx* ctx);

/* ---- stochastic dynamic adhesion model (section 3.2, Eq. 12-14, rules
 * L147-149, P_f / P_r L151) and short-range wall repulsion (section 3.4.1); the step
 * after S5 in the paper's loop (L276).  Readings A-1 .. A-9 in DESIGN.md.  Lattice units, rates
 * per time step.
 *   receptors : receptor r sits on global node h_node[r] (Eq. 14: "bond located at ith node");
 *   vWF sites : on the LOW face of wall axis `wall_axis` (the paper's "bottom plane"), one per
 *               lattice point of that plane (25 per um^2 = one per h^2 at h = 0.2 um, L145, L173).
 *               The plane lies at -1/2 (PLB_WALL_BB) or 0 (PLB_WALL_HH).  A site is named by its two
 *               tangential integer coordinates (s0, s1), tangential axes in x, y, z order, kept
 *               unwrapped like the node positions;
 *   k_on  = k_on0  exp( s d (gamma - d/2) ),  d = |x_b - l_b|,  s = sigma / k_B T        (Eq. 13)
 *   k_off = k_off0 exp( gamma s d )            (Eq. 12, Bell, with F_b = sigma d)
 *   P_f = 1 - exp(-k_on),  P_r = 1 - exp(-k_off)                                        (L151)
 *   bond force on its node : sigma (x_b - l_b) (S - X)/x_b   (Eq. 14 read as the restoring force)
 *   repulsion on every node: F0 tau exp(-tau eps)/(1 - exp(-tau eps)) along the inward normal,
 *               eps = distance of the node from the wall plane (L246); eps <= 0 raises the
 *               PLB_ERR_NODE_LEFT flag.                                                         */
typedef struct {
    int   wall_axis;      /* 0, 1, 2: must be a wall axis of the context */
    int   max_per_site;   /* rule 2 (L148): 4; at most 32 */
    float k_on0, k_off0;
    float s;              /* sigma / k_B T */
    float gamma;          /* reactive compliance (a length) */
    float sigma;          /* bond spring constant */
    float l_b, l_max;     /* equilibrium bond length; capture distance (128 nm = 0.64 h, L149) */
    float F0, tau_rep;    /* repulsion; F0 = 0 switches it off */
} plb_adhesion;

/* Device bytes ib_set_receptors needs for n_receptors receptors on this grid and wall axis. */
PLB_API int ib_adhesion_workspace_bytes(const plb_grid* grid, int wall_axis, long n_receptors, size_t* out_bytes);
/* Attach the receptors (all meshes must have been added).  d_workspace: caller-owned, 256-byte
 * aligned, ib_adhesion_workspace_bytes() bytes, valid until lbm_destroy.  All bonds start open.
 * From then on ib_compute_membrane_forces adds the bond and repulsion forces. */
PLB_API int ib_set_receptors(plb_ctx* ctx, long n_receptors, const int* h_node, const plb_adhesion* prm,
                     void* d_workspace, size_t workspace_bytes);
/* One Monte-Carlo update at the current node positions (call it after ib_interpolate_advance):
 * every existing bond is tested for breakage, then every unbound receptor whose nearest vWF site
 * is closer than l_max is tested for formation (order of L276).  Uniforms from Philox keyed on
 * (seed; receptor, step, tag 3): word 0 breaks (u < P_r), word 1 forms (u < P_f).  Probabilities
 * are evaluated in fp64.  When more receptors pass the formation test for one site than it has
 * free places, the lowest receptor indices take them (any number of same-step candidates). */
PLB_API int ib_adhesion_update(plb_ctx* ctx, unsigned long long seed, unsigned long long step);
PLB_API int ib_n_receptors(plb_ctx* ctx, long* out);
/* h_bonds: 3 ints per receptor = (bound 0/1, s0, s1) */
PLB_API int ib_read_bonds(plb_ctx* ctx, int* h_bonds);
PLB_API int ib_write_bonds(plb_ctx* ctx, const int* h_bonds);   /* also rebuilds the per-site counts */

/* ---- auxiliary, off the timed path (tests, checkpoints, end-to-end I/O) ---- */
PLB_API int ib_n_nodes(plb_ctx* ctx, long* out);
PLB_API int ib_read_nodes(plb_ctx* ctx, double* h_xyz);            /* n x 3 AoS */
PLB_API int ib_write_nodes(plb_ctx* ctx, const double* h_xyz);
PLB_API int ib_read_forces(plb_ctx* ctx, float* h_F);              /* n x 3 AoS */
PLB_API int ib_write_forces(plb_ctx* ctx, const float* h_F);       /* marks forces valid (tests) */
PLB_API int ib_read_node_velocities(plb_ctx* ctx, float* h_U);     /* n x 3 AoS, of the last interpolate */
/* populations in the paper's order, true f_i (not the stored f_i - w_i), float[19*cells] SoA */
PLB_API int lbm_read_populations(plb_ctx* ctx, float* d_f);
PLB_API int lbm_write_populations(plb_ctx* ctx, const float* d_f);
/* debug aid: number of cells of the current state (what lbm_read_macros sees) with a non-finite
 * population or a density sum_i f_i (Eq. 17) that is not positive (0 = healthy); synchronises the
 * stream */
PLB_API int lbm_check_finite(plb_ctx* ctx, long* out_bad_cells);
/* The same count (Eq. 17: density = sum_i f_i; SURVEY.md section 5 debug aid) for
 * callers that can neither allocate nor synchronise at the point of the call (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc): the scratch of the reduction is a
 * file-scope device array inside the library -- 256 KiB, held by every GPU that loads libplb.so until
 * the process exits -- and the call allocates nothing, copies nothing and does not wait.
 *   d_out_bad_cells : DEVICE pointer to one int (caller-owned); written asynchronously on the
 *                     context's stream with the number of bad cells (deterministic, no atomics).
 * Grids of more than PLB_STATIC_MAX_CELLS cells are refused with PLB_ERR_WORKSPACE; PLB_ERR_ORDER
 * before the populations were set; PLB_ERR_ARG for a null pointer.  All calls on one device share
 * the scratch array: calls that overlap on the GPU (other streams, other contexts) RACE on it;
 * calls on one stream are safe back to back. */
#define PLB_STATIC_MAX_CELLS 16777216L
PLB_API int lbm_check_finite_static(plb_ctx* ctx, int* d_out_bad_cells);
/* synchronise the stream; returns PLB_ERR_NODE_LEFT / PLB_ERR_CUDA if raised since creation */
PLB_API int plb_status(plb_ctx* ctx);
/* number of kernels this context has launched so far (for gpu_launches accounting) */
PLB_API int plb_launch_count(plb_ctx* ctx, long* out);
/* Philox4x32-10 block function on the device, for the known-answer test:
 * d_ctr uint32[4n], d_key uint32[2n] -> d_out uint32[4n] */
PLB_API int plb_philox4x32_10(void* cuda_stream, long n, const unsigned* d_ctr, const unsigned* d_key,
                      unsigned* d_out);

#ifdef __cplusplus
}
#endif
#endif
