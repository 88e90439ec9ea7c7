// plb_internal.cuh -- device helpers and host context shared by the libplb translation units.
// (Nothing here is shared with oracle/: the CPU oracle is an independent implementation.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <vector>
#include "../../include/plb.h"

namespace plb {

constexpr int Q = 19;
// Activity segments: 8 consecutive cells (one 128-byte line of the float4 forcing field, one
// 32-byte sector of a population row).  Bit (s & 31) of seg_mask[s >> 5] is set while segment s
// holds spread force.
#ifndef PLB_SEG_SHIFT
#define PLB_SEG_SHIFT 3
#endif
constexpr int SEG_SHIFT = PLB_SEG_SHIFT;
constexpr int SEG = 1 << SEG_SHIFT;

// D3Q19 velocity set in the paper's numbering (Eq. 21, Eq. 23-30; index = paper's i - 1).
__host__ __device__ constexpr int CX(int d) {
    constexpr int t[Q] = {1, -1, 0, 0, 0, 0, 1, 1, 1, 1, -1, -1, -1, -1, 0, 0, 0, 0, 0};
    return t[d];
}
__host__ __device__ constexpr int CY(int d) {
    constexpr int t[Q] = {0, 0, 1, -1, 0, 0, 1, -1, 0, 0, 1, -1, 0, 0, 1, 1, -1, -1, 0};
    return t[d];
}
__host__ __device__ constexpr int CZ(int d) {
    constexpr int t[Q] = {0, 0, 0, 0, 1, -1, 0, 0, 1, -1, 0, 0, 1, -1, 1, -1, 1, -1, 0};
    return t[d];
}
__host__ __device__ constexpr int OPP(int d) {
    constexpr int t[Q] = {1, 0, 3, 2, 5, 4, 11, 10, 13, 12, 7, 6, 9, 8, 17, 16, 15, 14, 18};
    return t[d];
}
__host__ __device__ constexpr float WGT(int d) {
    return d < 6 ? (1.0f / 18.0f) : (d < 18 ? (1.0f / 36.0f) : (1.0f / 3.0f));
}

struct LbmParams {
    int nx, ny, nz;
    int cells;                 // nx*ny*nz < 2^31
    int wall[3];               // boundary kind of the axis: PLB_PERIODIC, PLB_WALL_BB or PLB_WALL_HH
    float omega;               // 1/tau
    float pref;                // 1 - 1/(2 tau)
    float corr[3][2][Q];       // [axis][0 = low face, 1 = high face][d] = 6 w_d (c_d . u_wall)
    float uw[3][2][3];         // [axis][face] wall velocity (on-site velocity walls)
};

// one constrained mesh (Eq. 4-5): its triangles [tri_first, tri_first + tri_count), a reference
// node for the fp64 relative coordinates, the unstressed totals and the three coefficients
struct MeshConstraint {
    int tri_first, tri_count, node_first, pad;
    double S0_tot, V0;
    float k_s, k_t, k_v, pad2;
};

// Pitches of the spread kernel's shared-memory tile (ib.cu): a row pitch = 4 (mod 8) words puts the
// 4 x 4 cells one node touches per instruction (4 consecutive x in 4 rows) into 16 different banks.
__host__ __device__ inline int tile_row_pitch(const int e0) { return e0 + ((4 - (e0 & 7)) & 7); }
// A plane pitch = 8 (mod 16) words puts the second half-warp of the binned spread (same 4 x 4 cells,
// two planes further) into the other 16 banks.
__host__ __device__ inline int tile_plane_pitch(const int row_pitch, const int e1) {
    const int r = row_pitch * e1;
    return r + ((8 - (r & 15)) & 15);
}

enum ForceMode { FORCE_NONE = 0, FORCE_DENSE = 1, FORCE_SPARSE = 2 };
enum InterpForm { PLB_INTERP_AUTO = 0, PLB_INTERP_TILE = 1, PLB_INTERP_DIRECT = 2, PLB_INTERP_PULL = 3 };

// consecutive meshes that share one spring table: nodes [node_first, node_first + n_meshes * nn)
struct SpringGroup {
    int node_first, n_meshes, nn, off_first;
    float k;
};
struct SpringGroupHost {
    int nn;
    float k;
    std::vector<float> rest;
    std::vector<int> edges;
};

// status bits raised by kernels (sticky)
enum { STATUS_NODE_LEFT = 1, STATUS_ZERO_EDGE = 2, STATUS_ADH_BAD_SITE = 8 };

// NEXT-4 (section 3.2 / 3.4.1): adhesion parameters as the kernels take them.  a = wall
// axis, (t0, t1) the tangential axes in x, y, z order, (n0, n1) their sizes = the vWF site grid,
// plane = position of the wall plane on axis a.  Decision arithmetic is fp64 (adhesion.cu).
constexpr int ADH_MAX_PER_SITE = 32;        // bound on plb_adhesion.max_per_site = rounds of the arbitration
constexpr int ADH_NO_OFFER = 0x7f7f7f7f;    // site_min of a site nobody offers to (memset 0x7f)
struct AdhParams {
    int a, t0, t1, n0, n1, per0, per1, max_per_site;
    double plane, k_on0, k_off0, s, gamma, sigma, l_b, l_max, F0, tau_rep;
};

__device__ __forceinline__ bool seg_active(const unsigned* __restrict__ seg_mask, const int cell) {
    return (__ldg(seg_mask + (cell >> (SEG_SHIFT + 5))) >> ((cell >> SEG_SHIFT) & 31)) & 1u;
}

// ---------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), written from the paper's description.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k) {
    constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(M0, c.x), lo0 = M0 * c.x;
        const uint32_t hi1 = __umulhi(M1, c.z), lo1 = M1 * c.z;
        c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
        k.x += W0;
        k.y += W1;
    }
    return c;
}
// xi = ((r >> 8) + 1/2) 2^-24, exact in fp32, never 0 or 1
__device__ __forceinline__ float uniform01(uint32_t r) {
    return ((float)(r >> 8) + 0.5f) * (1.0f / 16777216.0f);
}
__device__ __forceinline__ uint4 noise_words(unsigned long long seed, unsigned long long index,
                                             uint32_t step, uint32_t tag) {
    return philox4x32_10(make_uint4((uint32_t)index, (uint32_t)(index >> 32), step, tag),
                         make_uint2((uint32_t)seed, (uint32_t)(seed >> 32)));
}

// ---------------------------------------------------------------------------------------------
// host context
// ---------------------------------------------------------------------------------------------
struct Ctx {
    plb_grid grid;
    float tau;
    plb_boundary bnd;
    LbmParams prm;
    cudaStream_t stream;
    long n_segs;
    // lattice (carved from the workspace)
    float* f[2];
    int cur;
    unsigned* seg_mask;        // one bit per segment, (n_segs + 31) / 32 words
    int* counters;             // [1] status bits, [2], [3] lengths of the segment list (alternating)
    int* seg_list;             // segments the last spread marked (n_segs entries)
    float4* vfield;            // (vx, vy, vz, rho) per cell, valid in the listed segments after segment_macros_kernel
    int list_parity;           // which counter the next spread appends to
    // meshes
    long cap_nodes, cap_edges, n_nodes, n_edges;
    double* X[3];              // SoA fp64 unwrapped positions
    float4* F;                 // nodal forces (Fx, Fy, Fz, 0)
    float4* U;                 // nodal velocities of the last interpolate
    double* stage;             // 3 * cap_nodes: AoS staging for ib_read_nodes / ib_write_nodes
    int* orig;                 // caller's global index of each stored node (the stored order is internal)
    std::vector<int> h_orig;   // the same on the host, and its inverse: h_stored[caller's index] = stored index
    std::vector<int> h_stored;
    // springs (Eq. 2-3): one table per topology, shared by all meshes of a group
    int* csr_off;              // rows: first entry of each local node (+ one end entry per table), global entry indices
    int2* csr_ent;             // entries: (neighbour's stored local index, rest length as float bits)
    long n_csr_off, n_csr_ent;
    std::vector<SpringGroup> groups;
    std::vector<SpringGroupHost> group_src;   // what each group was built from (to recognise a repeat)
    std::vector<long> mesh_node_off, mesh_edge_off;
    // area / volume constraints (Eq. 4-5): triangles of the constrained meshes, mesh by mesh
    long cap_tris, n_tris;
    int4* tris;                // (a, b, c, 0) global node indices, outward orientation
    float* tri_S0;             // unstressed triangle area
    MeshConstraint* cons;      // one entry per constrained mesh = one thread block of the kernel
    long cap_cons, n_cons;
    std::vector<char> mesh_constrained;
    int2* ranges;              // node ranges [first, last) served by one thread block of the IB kernels
    long n_ranges;
    int* range_box;            // per range: min and max of floor(X) as the last spread saw them (8 ints), first box_cap ranges
    int box_cap;
    int tile_cap;              // cells of the shared-memory lattice tile of the interpolation kernel
    int spread_cap;            // words per component of the (padded, bank-conflict-free) spread tile
    int interp_form;           // PLB_INTERP_*: AUTO, or the form forced through the PLB_INTERP environment variable
    int range_nodes;           // > 0: nodes per IB thread block forced through PLB_RANGE_NODES
    int spread_mode;           // PLB_SPREAD_*: which form of the spread kernel runs (AUTO: by tile_density)
    double tile_nodes, tile_cells;   // sums over the ranges at ib_add_meshes time: nodes, cells of their tiles
    double tile_density;       // tile_nodes / tile_cells
    // NEXT-4: receptors and bonds (carved from the caller's adhesion workspace)
    bool adh_on;
    AdhParams adh;
    long n_rec;
    int* rec_node;             // global node of each receptor
    int4* bond;                // (bound, s0, s1, candidate site of the running update or -1)
    int* site_count;           // bonds per vWF site, n0 * n1
    int* site_min;             // lowest receptor index among the pending candidates of a site (ADH_NO_OFFER: none)
    // bookkeeping
    const float4* g_last;
    int g_last_mode;           // ForceMode used by the last lbm_step
    float4* spread_target;     // buffer ib_spread last filled (its touched cells are listed in seg_list)
    bool spread_current;       // seg_list matches the current node positions
    bool listed_all;           // the last spread listed every stencil cell (not only the cells that received force)
    bool forces_valid;
    bool populated;
    long launches;
    int sm_count;
};

void set_error(const char* fmt, ...);
int cuda_check(cudaError_t e, const char* what);

// kernels launchers (lbm.cu / ib.cu); all asynchronous on c->stream, return a PLB_* code
int launch_set_equilibrium(Ctx* c, const float* d_rho, const float* d_u, float amp, unsigned long long seed);
int launch_lbm_step(Ctx* c, const float4* g, int mode);
int launch_read_macros(Ctx* c, float* d_rho, float* d_u);
int launch_read_populations(Ctx* c, float* d_f);
int launch_check_finite(Ctx* c, int* d_bad);
int launch_check_finite_static(Ctx* c, int* d_out);
int launch_write_populations(Ctx* c, const float* d_f);
int launch_membrane_forces(Ctx* c, float sigma, unsigned long long seed, unsigned long long step);
// host-side geometry of the unstressed shape (set-up, not on the timed path)
void reference_area_volume(const double* xyz, int n_tris, const int* tris, float* S0, double* S0_tot, double* V0);
int launch_clear_spread(Ctx* c, float4* g);
int launch_spread(Ctx* c, float4* g, bool after_clear);
int spread_mode_of(const Ctx* c);
int interp_form_of(const Ctx* c);
int launch_interpolate_advance(Ctx* c);
int ib_max_tile_cap();
int ib_max_spread_cap();
int launch_nodes_transpose(Ctx* c, bool to_aos);
int launch_adhesion_forces(Ctx* c);
int launch_adhesion_update(Ctx* c, unsigned long long seed, unsigned long long step);
int launch_adhesion_recount(Ctx* c);
int launch_philox(cudaStream_t s, long n, const unsigned* ctr, const unsigned* key, unsigned* out);

}  // namespace plb

struct plb_ctx : plb::Ctx {};
