// ib.cu -- immersed-boundary and membrane kernels (Eq. 2-3, section 3.4.2 Eq. 31-36).
//
// Node data: positions SoA fp64 (unwrapped), forces / node velocities float4 AoS.
// The forcing field is float4 per cell so that the spread ends in one 128-bit vector atomic per
// touched tile cell (red.global.add.v4.f32, sm_90+).  The nodes of a mesh are stored along the
// Morton curve of the mesh's initial shape (api.cu); `orig` maps a stored node to the caller's index.
#include <climits>
#include "plb_internal.cuh"
#include "lbm_device.cuh"

namespace plb {

// ---------------------------------------------------------------------------------------------
// S1: Hookean spring forces (Eq. 2-3) as a GATHER: one thread per node sums
//     F_i = sum_j k (|R| - L_ij) R/|R|,  R = X_j - X_i,  over its neighbours j
// (the force on i of Eq. 3 with the sign of DESIGN.md G1; an edge is evaluated from both ends).
// The topology is fixed and shared by all meshes of a group, so the (neighbour, rest length) table
// is stored ONCE per topology (123 KB for a 2562-node platelet: it lives in L1/L2) and the kernel
// streams only the positions and the forces: 24 B read + 16 B written per node instead of the
// 12 B per edge + 2 x 16 B atomics of an edge-parallel scatter; no zero-fill pass, no atomics, a
// fixed summation order (deterministic).  The hidden Morton order of the nodes keeps a node's
// neighbours within a few sectors of it.
// R and |R| - L are formed in fp64 (positions reach ~1e3, lengths ~1, stretches ~1e-3): 1/|R| is
// an fp32 rsqrt refined by one Newton step in fp64 (error ~1e-13), not a division and a square
// root.  Optional per-node noise (config 5): Box-Muller on Philox keyed on the caller's node index.
// ---------------------------------------------------------------------------------------------
// 1: Box-Muller through the hardware approximations (config 5: 0.610 -> 0.582 ms); 0: libm accuracy
#ifndef PLB_FAST_NOISE
#define PLB_FAST_NOISE 1
#endif
#ifndef PLB_FORCE_MINB
#define PLB_FORCE_MINB 5
#endif
__global__ void __launch_bounds__(256, PLB_FORCE_MINB) node_force_kernel(const double* __restrict__ X, const double* __restrict__ Y,
                                                         const double* __restrict__ Z, const int* __restrict__ orig,
                                                         const int* __restrict__ csr_off, const int2* __restrict__ csr_ent,
                                                         float4* __restrict__ F, const SpringGroup grp, const float sigma,
                                                         const unsigned long long seed, const unsigned step,
                                                         int* __restrict__ counters) {
    const long t = blockIdx.x * 256L + threadIdx.x;
    if (t >= (long)grp.n_meshes * grp.nn) return;
    const int local = (int)(t % grp.nn);
    const int base = grp.node_first + (int)(t - local);               // first node of this node's mesh
    const int m = base + local;
    const double xi = X[m], yi = Y[m], zi = Z[m];
    float4 f = make_float4(0.f, 0.f, 0.f, 0.f);
    const int e0 = __ldg(csr_off + grp.off_first + local), e1 = __ldg(csr_off + grp.off_first + local + 1);
    // (one neighbour at a time: batching the loads of a node's 6 neighbours -- 64 to 96 registers --
    // cost more in occupancy than it gained in latency: 0.64 to 1.08 ms against 0.61 ms at config 5)
    for (int e = e0; e < e1; ++e) {
        const int2 ent = __ldg(csr_ent + e);
        const int j = base + ent.x;
        const double rx = X[j] - xi, ry = Y[j] - yi, rz = Z[j] - zi;
        const double l2 = rx * rx + ry * ry + rz * rz;
        if (!(l2 > 0.0)) {
            atomicOr(counters + 1, STATUS_ZERO_EDGE);
            continue;
        }
        const float l2f = (float)l2;
        double r;                                                     // 1/|R|
        if (l2f > 1e-30f && l2f < 1e30f) {
            r = (double)rsqrtf(l2f);
            r = r * (1.5 - 0.5 * l2 * r * r);
        } else {
            r = 1.0 / sqrt(l2);
        }
        const float s = grp.k * (float)((l2 * r - (double)__int_as_float(ent.y)) * r);
        f.x = fmaf(s, (float)rx, f.x);
        f.y = fmaf(s, (float)ry, f.y);
        f.z = fmaf(s, (float)rz, f.z);
    }
    if (sigma > 0.f) {
        // Box-Muller on the four uniforms of counter (node, step, tag 2); the key is the caller's
        // global node index, not the stored one
        const uint4 r = noise_words(seed, (unsigned long long)__ldg(orig + m), step, 2u);
#if PLB_FAST_NOISE
        // hardware approximations (MUFU.LG2 / SIN / COS, absolute error ~4e-7 on log and on sin, cos):
        // the noise term moves by < 1e-6 sigma.  The angle is reduced to (-pi, pi] first.
        const float r0 = sqrtf(-2.0f * __logf(uniform01(r.x)));
        const float r2 = sqrtf(-2.0f * __logf(uniform01(r.z)));
        const float a1 = 6.283185307f * (uniform01(r.y) - (uniform01(r.y) > 0.5f ? 1.0f : 0.0f));
        const float a2 = 6.283185307f * (uniform01(r.w) - (uniform01(r.w) > 0.5f ? 1.0f : 0.0f));
        f.x += sigma * r0 * __cosf(a1);
        f.y += sigma * r0 * __sinf(a1);
        f.z += sigma * r2 * __cosf(a2);
#else
        const float r0 = sqrtf(-2.0f * logf(uniform01(r.x)));
        const float r2 = sqrtf(-2.0f * logf(uniform01(r.z)));
        float s1, c1;
        sincospif(2.0f * uniform01(r.y), &s1, &c1);
        f.x += sigma * r0 * c1;
        f.y += sigma * r0 * s1;
        f.z += sigma * r2 * cospif(2.0f * uniform01(r.w));
#endif
    }
    F[m] = f;
}

// ---------------------------------------------------------------------------------------------
// S1b: area and volume constraint forces, Eq. 4-5 (L101-108):
//   H = k_s (S_tot - S0_tot)^2/(2 S0_tot) + sum_tri k_t (S - S_0)^2/(2 S_0) + k_v (V - V_0)^2/(2 V_0)
//   S = |n|/2, n = (X_b - X_a) x (X_c - X_a);  V = (1/6) sum_tri X_a . (X_b x X_c)
//   F_a -= [k_s (S_tot - S0_tot)/S0_tot + k_t (S - S_0)/S_0] (1/2) nhat x (X_c - X_b)
//          + k_v (V - V_0)/V_0 (1/6) X_b x X_c                     (cyclic in a, b, c)
// One thread block per constrained mesh: pass 1 reduces S_tot and V over the mesh's triangles in
// a fixed order (deterministic), pass 2 scatters the forces (one vector atomic per corner).
// Geometry in fp64 relative to the mesh's first node (positions reach ~1e3, S - S_0 ~ 1e-3 S;
// V and its gradient summed over a closed surface do not depend on the origin).
// ---------------------------------------------------------------------------------------------
constexpr int CON_THREADS = 256;

struct TriGeom {
    double ax, ay, az, bx, by, bz, cx, cy, cz;   // corners relative to the reference node
    double nx, ny, nz, len;                      // n = (b - a) x (c - a), |n|
};

__device__ __forceinline__ TriGeom tri_geom(const double* __restrict__ X, const double* __restrict__ Y,
                                            const double* __restrict__ Z, const int4 t, const double ox,
                                            const double oy, const double oz) {
    TriGeom g;
    g.ax = __ldg(X + t.x) - ox; g.ay = __ldg(Y + t.x) - oy; g.az = __ldg(Z + t.x) - oz;
    g.bx = __ldg(X + t.y) - ox; g.by = __ldg(Y + t.y) - oy; g.bz = __ldg(Z + t.y) - oz;
    g.cx = __ldg(X + t.z) - ox; g.cy = __ldg(Y + t.z) - oy; g.cz = __ldg(Z + t.z) - oz;
    const double ux = g.bx - g.ax, uy = g.by - g.ay, uz = g.bz - g.az;
    const double vx = g.cx - g.ax, vy = g.cy - g.ay, vz = g.cz - g.az;
    g.nx = uy * vz - uz * vy; g.ny = uz * vx - ux * vz; g.nz = ux * vy - uy * vx;
    g.len = sqrt(g.nx * g.nx + g.ny * g.ny + g.nz * g.nz);
    return g;
}

__device__ __forceinline__ double block_sum(double v, double* scratch) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) scratch[threadIdx.x >> 5] = v;
    __syncthreads();
    double tot = 0.0;
#pragma unroll
    for (int w = 0; w < CON_THREADS / 32; ++w) tot += scratch[w];
    return tot;
}

__global__ void __launch_bounds__(CON_THREADS) constraint_force_kernel(
    const double* __restrict__ X, const double* __restrict__ Y, const double* __restrict__ Z,
    const int4* __restrict__ tris, const float* __restrict__ tri_S0, const MeshConstraint* __restrict__ cons,
    float4* __restrict__ F) {
    __shared__ double scratch[CON_THREADS / 32];
    const MeshConstraint m = cons[blockIdx.x];
    const double ox = __ldg(X + m.node_first), oy = __ldg(Y + m.node_first), oz = __ldg(Z + m.node_first);
    double S = 0.0, V6 = 0.0;
    for (int t = threadIdx.x; t < m.tri_count; t += CON_THREADS) {
        const TriGeom g = tri_geom(X, Y, Z, __ldg(tris + m.tri_first + t), ox, oy, oz);
        S += 0.5 * g.len;
        V6 += g.ax * (g.by * g.cz - g.bz * g.cy) + g.ay * (g.bz * g.cx - g.bx * g.cz) + g.az * (g.bx * g.cy - g.by * g.cx);
    }
    const double S_tot = block_sum(S, scratch);
    const double V = block_sum(V6, scratch) * (1.0 / 6.0);
    const double alpha = (double)m.k_s * (S_tot - m.S0_tot) / m.S0_tot;
    const double beta6 = (double)m.k_v * (V - m.V0) / m.V0 * (1.0 / 6.0);
    for (int t = threadIdx.x; t < m.tri_count; t += CON_THREADS) {
        const int4 tv = __ldg(tris + m.tri_first + t);
        const TriGeom g = tri_geom(X, Y, Z, tv, ox, oy, oz);
        const double S0 = (double)__ldg(tri_S0 + m.tri_first + t);
        const double inv = g.len > 0.0 ? 1.0 / g.len : 0.0;
        const double hx = g.nx * inv, hy = g.ny * inv, hz = g.nz * inv;            // nhat
        const double cS = 0.5 * (alpha + (double)m.k_t * (0.5 * g.len - S0) / S0);
        // corner a: nhat x (c - b), b x c;  corner b: nhat x (a - c), c x a;  corner c: nhat x (b - a), a x b
        double ex = g.cx - g.bx, ey = g.cy - g.by, ez = g.cz - g.bz;
        atomicAdd(F + tv.x, make_float4(
            (float)-(cS * (hy * ez - hz * ey) + beta6 * (g.by * g.cz - g.bz * g.cy)),
            (float)-(cS * (hz * ex - hx * ez) + beta6 * (g.bz * g.cx - g.bx * g.cz)),
            (float)-(cS * (hx * ey - hy * ex) + beta6 * (g.bx * g.cy - g.by * g.cx)), 0.f));
        ex = g.ax - g.cx; ey = g.ay - g.cy; ez = g.az - g.cz;
        atomicAdd(F + tv.y, make_float4(
            (float)-(cS * (hy * ez - hz * ey) + beta6 * (g.cy * g.az - g.cz * g.ay)),
            (float)-(cS * (hz * ex - hx * ez) + beta6 * (g.cz * g.ax - g.cx * g.az)),
            (float)-(cS * (hx * ey - hy * ex) + beta6 * (g.cx * g.ay - g.cy * g.ax)), 0.f));
        ex = g.bx - g.ax; ey = g.by - g.ay; ez = g.bz - g.az;
        atomicAdd(F + tv.z, make_float4(
            (float)-(cS * (hy * ez - hz * ey) + beta6 * (g.ay * g.bz - g.az * g.by)),
            (float)-(cS * (hz * ex - hx * ez) + beta6 * (g.az * g.bx - g.ax * g.bz)),
            (float)-(cS * (hx * ey - hy * ex) + beta6 * (g.ax * g.by - g.ay * g.bx)), 0.f));
    }
}

// ---------------------------------------------------------------------------------------------
// 4-point cosine delta (Eq. 36): for a node at X, base = floor(X) - 1, frac = X - floor(X),
// the four weights at cells base + o are phi(frac + 1 - o):
//     o=0: (1 - s)/4   o=1: (1 + c)/4   o=2: (1 + s)/4   o=3: (1 - c)/4,
// s = sin(pi frac/2), c = cos(pi frac/2)   (cos(a + pi/2) = -sin a, cos(a - pi) = -cos a).
// ---------------------------------------------------------------------------------------------
// wrapped index on a periodic axis; -1 if dropped on a wall axis
__device__ __forceinline__ int wrap_index(int q, const int n, const int wall) {
    if (q >= 0 && q < n) return q;
    if (wall) return -1;
    q %= n;
    return q < 0 ? q + n : q;
}

// ---------------------------------------------------------------------------------------------
// S2 and S4/S5 run one thread block per NODE RANGE: a mesh, or a run of consecutive stored nodes of
// a mesh (a surface patch, thanks to the hidden Morton order) when there are few meshes or a mesh is
// very large.  A platelet is a compact object: the 4x4x4 supports of its nodes overlap heavily (about
// 13 contributions per touched cell at config 4, 1000 at config 5), so the block accumulates /
// gathers through a TILE of the lattice held in shared memory -- the bounding box of the
// supports of its nodes -- and touches global memory once per tile cell:
//   spread:       zero tile -> nodes scatter into the tile -> the non-zero tile cells go to the
//                 forcing field with one 128-bit RED each.  The tile accumulates in 32-bit fixed
//                 point with a per-block power-of-two scale (native shared-memory integer
//                 atomics; the fp32 ones are compare-and-swap loops): order-independent, and
//                 with a resolution of n_nodes/8 * 2^-30 of the largest nodal force component;
//   interpolate:  (pull form) mark the tile cells some node needs -> compact them -> their v
//                 straight from the 19 pulled populations (no velocity field in HBM) -> nodes gather
//                 from the tile; (listed-cells form, densely sampled meshes) the velocity of every
//                 listed cell once, in a pre-pass -> tile copied from that field -> gather.
// A range whose bounding box does not fit the tile (a non-compact "mesh") takes the direct path:
// global REDs per (node, cell) and on-the-fly cell moments.  Both paths compute the same sums.
// Lane layouts (each measured against the alternatives on the B200):
//   interpolate:  FOUR lanes serve one node: lane = ox (the x offset of the stencil column), each
//                 lane walks the 4 x 4 (oy, oz) cells of its column; the lanes share the per-node
//                 set-up (lane a < 3 does floor / sincospi of axis a) and finish with a 4-lane
//                 shuffle reduction;
//   spread:       SIXTEEN lanes serve one node (lane = (ox, oy), loop over oz) from per-node records
//                 staged in shared memory (see spread_mesh_kernel).
// ---------------------------------------------------------------------------------------------
#ifndef PLB_IB_THREADS
#define PLB_IB_THREADS 512
#endif
constexpr int IB_THREADS = PLB_IB_THREADS;
constexpr int NODE_LANES = 4;
constexpr int SPREAD_SEG_LIST = 2048;   // segments one spread block can newly mark before it appends one by one
constexpr int IB_GROUPS = IB_THREADS / NODE_LANES;

struct MeshTile {
    int o[3];            // unwrapped lattice coordinate of tile cell (0,0,0)
    int e[3];            // extent in cells
    int p0, pp;          // row and plane pitch of the stored tile (= e[0], e[0] * e[1] unless padded)
    int lo[3], hi[3];    // tile coordinates [lo, hi) that exist on the lattice (wall axes clip)
    int enabled;
    int clipped;         // some [lo, hi) is smaller than the extent: stencils need the range check
    int interior;        // every tile cell and its 18 neighbours lie inside the grid: no wrap, no wall
    int mn[3], mx[3];    // reduction scratch: min / max of floor(X)
    unsigned fmax_bits;  // reduction scratch: largest |F| component (non-negative float bits)
    int n_need;          // interpolate: number of tile cells some node needs; spread: segments newly marked
};

// Programmatic dependent launch (sm_90+): ib_spread launches clear_spread_kernel and then the spread
// kernel.  The clear lets its dependent start at once (launch_dependents), and the spread kernel
// runs everything that does not touch what the clear writes -- bounding box, tile zeroing, the
// whole scatter into shared memory -- before it waits for the clear to have completed (wait),
// just ahead of its flush into the forcing field, the activity mask and the segment list.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// set the activity bit of the 8-cell segment of a cell; the thread that sets it first also appends
// the segment to the list the next ib_spread clears from
__device__ __forceinline__ void mark_segment(const int cell, unsigned* __restrict__ seg_mask, int* __restrict__ seg_list,
                                             int* __restrict__ seg_count) {
    const int seg = cell >> SEG_SHIFT;
    const unsigned bit = 1u << (seg & 31);
    unsigned* word = seg_mask + (seg >> 5);
    if ((*(volatile unsigned*)word & bit) == 0u) {
        if ((atomicOr(word, bit) & bit) == 0u) seg_list[atomicAdd(seg_count, 1)] = seg;
    }
}

// tile geometry from the box T.mn, T.mx of floor(X) over the range (one thread)
__device__ __forceinline__ void tile_geometry(MeshTile& T, const bool nonempty, const LbmParams& p, const int cap,
                                              const bool padded) {
    const int n[3] = {p.nx, p.ny, p.nz};
    long long vol = 1;
    bool ok = nonempty, clipped = false, interior = true;
    for (int a = 0; a < 3; ++a) {
        const long long ext = (long long)T.mx[a] - (long long)T.mn[a] + 4;
        ok = ok && ext <= (long long)cap;
        T.o[a] = T.mn[a] - 1;
        T.e[a] = ok ? (int)ext : 1;
        vol *= T.e[a];
        ok = ok && vol <= (long long)cap;
        if (p.wall[a] && ok) {
            const long long lo = -(long long)T.o[a], hi = (long long)n[a] - (long long)T.o[a];
            T.lo[a] = (int)max(0LL, min(lo, ext));
            T.hi[a] = (int)max(0LL, min(hi, ext));
        } else {
            T.lo[a] = 0; T.hi[a] = T.e[a];
        }
        clipped = clipped || T.lo[a] != 0 || T.hi[a] != T.e[a];
        interior = interior && (long long)T.o[a] >= 1 && (long long)T.o[a] + ext <= (long long)n[a] - 1;
    }
    T.p0 = padded ? tile_row_pitch(T.e[0]) : T.e[0];
    T.pp = padded ? tile_plane_pitch(T.p0, T.e[1]) : T.e[0] * T.e[1];
    ok = ok && (long long)T.pp * T.e[2] <= (long long)cap;
    T.enabled = ok ? 1 : 0;
    T.clipped = clipped ? 1 : 0;
    T.interior = (ok && interior) ? 1 : 0;
}

// bounding box of the supports of nodes [n0, n1) -> tile geometry (all threads of the block);
// with F != nullptr also the largest force component of the range; with box_out != nullptr the box
// is also stored (8 ints) for the interpolation of the same positions
__device__ __forceinline__ void tile_setup(MeshTile& T, const double* __restrict__ X, const double* __restrict__ Y,
                                           const double* __restrict__ Z, const float4* __restrict__ F, const int n0,
                                           const int n1, const LbmParams& p, const int cap, const bool padded,
                                           int* __restrict__ box_out = nullptr) {
    if (threadIdx.x == 0) {
        for (int a = 0; a < 3; ++a) { T.mn[a] = INT_MAX; T.mx[a] = INT_MIN; }
        T.fmax_bits = 0u;
        T.n_need = 0;
    }
    __syncthreads();
    int mn[3] = {INT_MAX, INT_MAX, INT_MAX}, mx[3] = {INT_MIN, INT_MIN, INT_MIN};
    float fmax = 0.f;
    for (int m = n0 + (int)threadIdx.x; m < n1; m += IB_THREADS) {
        const int f0 = (int)floor(X[m]), f1 = (int)floor(Y[m]), f2 = (int)floor(Z[m]);
        mn[0] = min(mn[0], f0); mx[0] = max(mx[0], f0);
        mn[1] = min(mn[1], f1); mx[1] = max(mx[1], f1);
        mn[2] = min(mn[2], f2); mx[2] = max(mx[2], f2);
        if (F) {
            const float4 f = __ldg(F + m);
            fmax = fmaxf(fmax, fmaxf(fabsf(f.x), fmaxf(fabsf(f.y), fabsf(f.z))));
        }
    }
    mn[0] = __reduce_min_sync(0xffffffffu, mn[0]); mx[0] = __reduce_max_sync(0xffffffffu, mx[0]);
    mn[1] = __reduce_min_sync(0xffffffffu, mn[1]); mx[1] = __reduce_max_sync(0xffffffffu, mx[1]);
    mn[2] = __reduce_min_sync(0xffffffffu, mn[2]); mx[2] = __reduce_max_sync(0xffffffffu, mx[2]);
    const unsigned fbits = __reduce_max_sync(0xffffffffu, __float_as_uint(fmax));
    if ((threadIdx.x & 31) == 0) {
        atomicMin(&T.mn[0], mn[0]); atomicMax(&T.mx[0], mx[0]);
        atomicMin(&T.mn[1], mn[1]); atomicMax(&T.mx[1], mx[1]);
        atomicMin(&T.mn[2], mn[2]); atomicMax(&T.mx[2], mx[2]);
        if (F) atomicMax(&T.fmax_bits, fbits);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        if (box_out) {
            box_out[0] = T.mn[0]; box_out[1] = T.mn[1]; box_out[2] = T.mn[2]; box_out[3] = n1 > n0 ? 1 : 0;
            box_out[4] = T.mx[0]; box_out[5] = T.mx[1]; box_out[6] = T.mx[2]; box_out[7] = 0;
        }
        tile_geometry(T, n1 > n0, p, cap, padded);
    }
    __syncthreads();
}

// tile cell index t -> (x, y, z) without integer division: t < 2^16 and 4 <= e0, e1 < 2^16, so
// floor(t / e) = umulhi(t, floor(2^32 / e) + 1) exactly (the error term t (m e - 2^32) / 2^32 stays
// below t e / 2^32 < 1).  The generic 32-bit division costs about 20 instructions, twice per cell.
struct TileSplit {
    unsigned m0, m1;
    int e0, e1;
    __device__ __forceinline__ explicit TileSplit(const MeshTile& T)
        : m0(0xffffffffu / (unsigned)T.e[0] + 1u), m1(0xffffffffu / (unsigned)T.e[1] + 1u), e0(T.e[0]), e1(T.e[1]) {}
    __device__ __forceinline__ void operator()(const int t, int& x, int& y, int& z) const {
        const int r = (int)__umulhi((unsigned)t, m0);
        x = t - r * e0;
        z = (int)__umulhi((unsigned)r, m1);
        y = r - z * e1;
    }
};

// global lattice cell of tile cell (x, y, z) (only called for cells inside [lo, hi) on wall axes)
__device__ __forceinline__ Cell tile_cell(const MeshTile& T, const int x, const int y, const int z, const LbmParams& p) {
    Cell c;
    c.i = wrap_index(T.o[0] + x, p.nx, 0);
    c.j = wrap_index(T.o[1] + y, p.ny, 0);
    c.k = wrap_index(T.o[2] + z, p.nz, 0);
    return c;
}

// The stencil of one node as its four lanes see it: lane `sub` owns the column ox = sub.
struct NodeStencil {
    int bx, by, bz;        // base = floor(X) - 1 per axis, minus `origin`
    float wx;              // weight of this lane's ox
    float wy[4], wz[4];    // weights of oy, oz = 0..3
};

// phi(frac + 1 - o), o = 0..3, from s = sin(pi frac/2), c = cos(pi frac/2)  (see weight_of)
__device__ __forceinline__ void weights4(const float s, const float c, float (&w)[4]) {
    w[0] = fmaf(-0.25f, s, 0.25f); w[1] = fmaf(0.25f, c, 0.25f);
    w[2] = fmaf(0.25f, s, 0.25f);  w[3] = fmaf(-0.25f, c, 0.25f);
}

// All 32 lanes call this; lane a < 3 of each 4-lane group holds x = coordinate a of the node (lane
// 3 a copy of X) and evaluates that axis (fp64 floor, sincospi of the fraction), then the group
// exchanges by shuffle.  The caller loads x one sweep ahead (node_coord) so that the global-load
// latency hides behind the previous sweep's shared-memory work.
__device__ __forceinline__ double node_coord(const double* X, const double* Y, const double* Z, const int m, const int sub) {
    const double* P = sub == 1 ? Y : (sub == 2 ? Z : X);
    return P[m];
}

template <bool WEIGHTS>
__device__ __forceinline__ NodeStencil node_stencil(const double x, const int sub, const int o0, const int o1, const int o2) {
    const double fl = floor(x);
    const int base = (int)fl - 1 - (sub == 1 ? o1 : (sub == 2 ? o2 : o0));
    float s = 0.f, c = 0.f;
    if (WEIGHTS) sincospif(0.5f * (float)(x - fl), &s, &c);
    NodeStencil st;
    st.bx = __shfl_sync(0xffffffffu, base, 0, NODE_LANES);
    st.by = __shfl_sync(0xffffffffu, base, 1, NODE_LANES);
    st.bz = __shfl_sync(0xffffffffu, base, 2, NODE_LANES);
    if (WEIGHTS) {
        const float sx = __shfl_sync(0xffffffffu, s, 0, NODE_LANES), cx = __shfl_sync(0xffffffffu, c, 0, NODE_LANES);
        const float sy = __shfl_sync(0xffffffffu, s, 1, NODE_LANES), cy = __shfl_sync(0xffffffffu, c, 1, NODE_LANES);
        const float sz = __shfl_sync(0xffffffffu, s, 2, NODE_LANES), cz = __shfl_sync(0xffffffffu, c, 2, NODE_LANES);
        const float t = (sub & 1) ? cx : sx;                       // o = 0: -s, 1: +c, 2: +s, 3: -c
        st.wx = fmaf((sub == 0 || sub == 3) ? -0.25f : 0.25f, t, 0.25f);
        weights4(sy, cy, st.wy);
        weights4(sz, cz, st.wz);
    }
    return st;
}

// S2: g_ijk += F_m phi phi phi (Eq. 34).  Also sets the activity bits of the touched segments.
// SIXTEEN lanes per node: lane = (ox, oy) walks the four oz cells of its stencil column.  The per-node
// set-up (fp64 floor, sincospi per axis, force scaling) is done once, one thread per node, for a
// chunk of 256 nodes at a time (coalesced loads, issued one chunk ahead) and staged in shared
// memory; the lanes read it back as broadcasts.  The tile is stored with a row pitch = 4 (mod 8)
// words, so the 16 cells a node touches per instruction fall into 16 different banks.
// (Measured on B200, config 4 / config 5: 4 lanes per node 0.136 / 2.44 ms, one warp per node with
// redundant set-up 0.124 / 2.87 ms; this layout is the fastest of the three.)
constexpr int SPREAD_LANES = 16;
constexpr int SPREAD_CHUNK = 256;
constexpr int SPREAD_GROUPS = IB_THREADS / SPREAD_LANES;

// phi(frac + 1 - o) from s = sin(pi frac/2), c = cos(pi frac/2): o = 0: (1 - s)/4, 1: (1 + c)/4,
// 2: (1 + s)/4, 3: (1 - c)/4
__device__ __forceinline__ float weight_o(const float s, const float c, const int o) {
    return fmaf((o == 0 || o == 3) ? -0.25f : 0.25f, (o & 1) ? c : s, 0.25f);
}

struct SpreadChunk {
    int* b;        // [3][SPREAD_CHUNK] base = floor(X) - 1 - tile origin
    float* sc;     // [6][SPREAD_CHUNK] sin, cos of pi frac/2 per axis
    float* f;      // [3][SPREAD_CHUNK] scaled force
};

__device__ __forceinline__ void spread_record(const SpreadChunk& ch, const int r, const double x, const double y,
                                              const double z, const float4 F, const float scale, const int o0,
                                              const int o1, const int o2) {
    const double fx = floor(x), fy = floor(y), fz = floor(z);
    ch.b[r] = (int)fx - 1 - o0;
    ch.b[SPREAD_CHUNK + r] = (int)fy - 1 - o1;
    ch.b[2 * SPREAD_CHUNK + r] = (int)fz - 1 - o2;
    float s, c;
    sincospif(0.5f * (float)(x - fx), &s, &c);
    ch.sc[r] = s; ch.sc[SPREAD_CHUNK + r] = c;
    sincospif(0.5f * (float)(y - fy), &s, &c);
    ch.sc[2 * SPREAD_CHUNK + r] = s; ch.sc[3 * SPREAD_CHUNK + r] = c;
    sincospif(0.5f * (float)(z - fz), &s, &c);
    ch.sc[4 * SPREAD_CHUNK + r] = s; ch.sc[5 * SPREAD_CHUNK + r] = c;
    ch.f[r] = F.x * scale; ch.f[SPREAD_CHUNK + r] = F.y * scale; ch.f[2 * SPREAD_CHUNK + r] = F.z * scale;
}

// Touched cells: a tile cell inside some node's stencil is LISTED (its segment marked) whatever its
// value, so that after ib_spread the segment list covers every cell the interpolation of the same
// positions will read -- also where the force is zero or rounds to zero.  Every node sets ONE bit,
// that of its base cell, in a bitmap with one 32-bit x-mask per (y, z) tile row; before the flush
// the bitmap is dilated by the 4 x 4 x 4 stencil (x by shifts, y and z by OR-ing 16 rows), one
// thread per row.  Tiles wider than 32 cells count every cell as touched.
__device__ __forceinline__ void touch_base(unsigned* __restrict__ binrow, const MeshTile& T, const int bx, const int by,
                                           const int bz) {
    unsigned* row = binrow + bz * T.e[1] + by;
    const unsigned bit = 1u << bx;
    if ((*(volatile unsigned*)row & bit) == 0u) atomicOr(row, bit);
}
// x cells of a tile row that lie on the lattice
__device__ __forceinline__ unsigned tile_exist_mask(const MeshTile& T) {
    const unsigned below_hi = T.hi[0] >= 32 ? 0xffffffffu : ((1u << T.hi[0]) - 1u);
    const unsigned below_lo = T.lo[0] >= 32 ? 0xffffffffu : ((1u << T.lo[0]) - 1u);
    return below_hi & ~below_lo;
}
// all threads of the block, after a __syncthreads(); followed by one
__device__ __forceinline__ void dilate_rows(const unsigned* __restrict__ binrow, unsigned* __restrict__ rowmask,
                                            const MeshTile& T) {
    const int e1 = T.e[1], e2 = T.e[2];
    const unsigned exist = tile_exist_mask(T);
    for (int r = threadIdx.x; r < e1 * e2; r += IB_THREADS) {
        const int y = r % e1, z = r / e1;
        unsigned m = 0u;
        if (y >= T.lo[1] && y < T.hi[1] && z >= T.lo[2] && z < T.hi[2]) {
            for (int bz = max(0, z - 3); bz <= z; ++bz)
                for (int by = max(0, y - 3); by <= y; ++by) m |= binrow[bz * e1 + by];
            m = (m | (m << 1) | (m << 2) | (m << 3)) & exist;
        }
        rowmask[r] = m;
    }
}

// Flush of a spread tile: one vector RED per non-zero tile cell.  The segments this block is the
// first to mark are collected in shared memory and appended to the global list with ONE atomicAdd
// per block (a returning atomic per segment on the single list counter was 58 % of the scatter
// kernel's stall samples).  All threads of the block call it, after a __syncthreads().
__device__ __forceinline__ void spread_flush(MeshTile& T, const int* __restrict__ tile, const unsigned* __restrict__ rowmask,
                                             const bool list_all, int* __restrict__ new_segs, const int cap,
                                             const float inv_scale, float4* __restrict__ g, unsigned* __restrict__ seg_mask,
                                             int* __restrict__ seg_list, int* __restrict__ seg_count, const LbmParams& p) {
    // list_all: every touched cell is listed (rowmask; a tile without row masks counts every existing
    // cell as touched); else only the cells that received force are (the interpolation will then not
    // rely on the list)
    const int tid = threadIdx.x;
    const int e1 = T.e[1], ncell = T.e[0] * e1 * T.e[2];
    const TileSplit split(T);
    for (int t = tid; t < ncell; t += IB_THREADS) {
        int x, y, z;
        split(t, x, y, z);
        const int w = z * T.pp + y * T.p0 + x;
        const int qx = tile[w], qy = tile[cap + w], qz = tile[2 * cap + w];
        const bool nonzero = (qx | qy | qz) != 0;
        bool listed = nonzero;
        if (list_all)
            listed = rowmask ? ((rowmask[z * e1 + y] >> x) & 1u) != 0u
                             : (x >= T.lo[0] && x < T.hi[0] && y >= T.lo[1] && y < T.hi[1] && z >= T.lo[2] && z < T.hi[2]);
        if (!listed) continue;
        const Cell c = tile_cell(T, x, y, z, p);
        const int cell = c.i + p.nx * (c.j + p.ny * c.k);
        if (nonzero)
            atomicAdd(g + cell, make_float4((float)qx * inv_scale, (float)qy * inv_scale, (float)qz * inv_scale, 0.f));
        const int seg = cell >> SEG_SHIFT;
        const unsigned bit = 1u << (seg & 31);
        unsigned* word = seg_mask + (seg >> 5);
        if ((*(volatile unsigned*)word & bit) == 0u && (atomicOr(word, bit) & bit) == 0u) {
            const int slot = atomicAdd(&T.n_need, 1);                   // n_need doubles as the block's list length
            if (slot < SPREAD_SEG_LIST) new_segs[slot] = seg;
            else seg_list[atomicAdd(seg_count, 1)] = seg;              // list full: append directly
        }
    }
    __syncthreads();
    const int n_new = min(T.n_need, SPREAD_SEG_LIST);
    if (n_new == 0) return;
    if (tid == 0) T.mn[0] = atomicAdd(seg_count, n_new);
    __syncthreads();
    const int first = T.mn[0];
    for (int i = tid; i < n_new; i += IB_THREADS) seg_list[first + i] = new_segs[i];
}

__global__ void __launch_bounds__(IB_THREADS, 1024 / IB_THREADS) spread_mesh_kernel(
    const double* __restrict__ X, const double* __restrict__ Y, const double* __restrict__ Z,
    const float4* __restrict__ F, const int2* __restrict__ ranges, float4* __restrict__ g,
    unsigned* __restrict__ seg_mask, int* __restrict__ seg_list, int* __restrict__ seg_count, const LbmParams p,
    const int cap, int* __restrict__ range_box, const int box_cap, const bool list_all) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ MeshTile T;
    int* tile = reinterpret_cast<int*>(smem_raw);                      // [3][cap] fixed point, padded pitches
    int* new_segs = tile + 3 * cap;                                    // [SPREAD_SEG_LIST]
    SpreadChunk ch;
    ch.b = new_segs + SPREAD_SEG_LIST;
    ch.sc = reinterpret_cast<float*>(ch.b + 3 * SPREAD_CHUNK);
    ch.f = ch.sc + 6 * SPREAD_CHUNK;
    unsigned* binrow = reinterpret_cast<unsigned*>(ch.f + 3 * SPREAD_CHUNK);    // [cap / 4] occupied base cells, x-mask per tile row
    unsigned* rowmask = binrow + cap / 4;                              // [cap / 4] touched cells, x-mask per tile row
    const int2 range = __ldg(ranges + blockIdx.x);
    const int n0 = range.x, n1 = range.y, tid = threadIdx.x;
    tile_setup(T, X, Y, Z, F, n0, n1, p, cap, true, (int)blockIdx.x < box_cap ? range_box + 8 * blockIdx.x : nullptr);
    const float fmax = __uint_as_float(T.fmax_bits);
    const bool tiled = T.enabled != 0 && fmax < 3.0e38f;
    if (!tiled) pdl_wait();                                            // the direct path writes the field as it goes
    const int nword = tiled ? T.pp * T.e[2] : 0;
    // |tile value| <= n_nodes * max W * max|F| = bound; scale = 2^k with bound * scale < 2^30
    // (a range without force still runs: its cells are listed for the interpolation)
    const int k = fmax > 0.f ? max(-100, min(100, 29 - ilogbf(0.125f * (float)(n1 - n0) * fmax))) : 0;
    const float scale = tiled ? ldexpf(1.0f, k) : 1.0f, inv_scale = ldexpf(1.0f, -k);
    for (int t = tid; t < nword; t += IB_THREADS) {
        tile[t] = 0; tile[cap + t] = 0; tile[2 * cap + t] = 0;
    }
    const bool by_rows = list_all && tiled && T.e[0] <= 32;
    if (by_rows)
        for (int t = tid; t < T.e[1] * T.e[2]; t += IB_THREADS) binrow[t] = 0u;
    const int sub = tid & (SPREAD_LANES - 1), ox = sub & 3, oy = sub >> 2, group = tid / SPREAD_LANES;
    const int o0 = tiled ? T.o[0] : 0, o1 = tiled ? T.o[1] : 0, o2 = tiled ? T.o[2] : 0;
    const int p0 = T.p0, pp = T.pp;
    const bool clipped = T.clipped != 0;
    // this thread's node of the coming chunk, loaded one chunk ahead
    double px = 0.0, py = 0.0, pz = 0.0;
    float4 pF = make_float4(0.f, 0.f, 0.f, 0.f);
    bool have = tid < SPREAD_CHUNK && n0 + tid < n1;
    if (have) { px = X[n0 + tid]; py = Y[n0 + tid]; pz = Z[n0 + tid]; pF = __ldg(F + n0 + tid); }
    for (int c0 = n0; c0 < n1; c0 += SPREAD_CHUNK) {
        __syncthreads();                                               // tile zeroed / previous chunk consumed
        if (have) {
            spread_record(ch, tid, px, py, pz, pF, scale, o0, o1, o2);
            if (by_rows) touch_base(binrow, T, ch.b[tid], ch.b[SPREAD_CHUNK + tid], ch.b[2 * SPREAD_CHUNK + tid]);
        }
        __syncthreads();
        const int m_next = c0 + SPREAD_CHUNK + tid;
        have = tid < SPREAD_CHUNK && m_next < n1;
        if (have) { px = X[m_next]; py = Y[m_next]; pz = Z[m_next]; pF = __ldg(F + m_next); }
        const int cnt = min(SPREAD_CHUNK, n1 - c0);
        for (int r = group; r < cnt; r += SPREAD_GROUPS) {
            const int bx = ch.b[r] + ox, by = ch.b[SPREAD_CHUNK + r] + oy, bz = ch.b[2 * SPREAD_CHUNK + r];
            const float wxy = weight_o(ch.sc[r], ch.sc[SPREAD_CHUNK + r], ox) *
                              weight_o(ch.sc[2 * SPREAD_CHUNK + r], ch.sc[3 * SPREAD_CHUNK + r], oy);
            const float sz = ch.sc[4 * SPREAD_CHUNK + r], cz = ch.sc[5 * SPREAD_CHUNK + r];
            const float fx = wxy * ch.f[r], fy = wxy * ch.f[SPREAD_CHUNK + r], fz = wxy * ch.f[2 * SPREAD_CHUNK + r];
            if (tiled) {
                if (clipped && (bx < T.lo[0] || bx >= T.hi[0] || by < T.lo[1] || by >= T.hi[1])) continue;
                const int t0 = bz * pp + by * p0 + bx;
#pragma unroll
                for (int oz = 0; oz < 4; ++oz) {
                    if (clipped && (bz + oz < T.lo[2] || bz + oz >= T.hi[2])) continue;
                    const float wz = weight_o(sz, cz, oz);
                    const int t = t0 + oz * pp;
                    // (F2I is not the limiter: the magic-number FMA of the gather form in its place
                    // changed nothing -- 0.0977 vs 0.0980 ms at config 4, 1.677 vs 1.692 ms at config 5)
                    atomicAdd(tile + t, __float2int_rn(wz * fx));
                    atomicAdd(tile + cap + t, __float2int_rn(wz * fy));
                    atomicAdd(tile + 2 * cap + t, __float2int_rn(wz * fz));
                }
            } else {
                const int qx = wrap_index(bx, p.nx, p.wall[0]), qy = wrap_index(by, p.ny, p.wall[1]);
                if (qx < 0 || qy < 0) continue;
#pragma unroll
                for (int oz = 0; oz < 4; ++oz) {
                    const int qz = wrap_index(bz + oz, p.nz, p.wall[2]);
                    if (qz < 0) continue;
                    const float wz = weight_o(sz, cz, oz);
                    const int cell = qx + p.nx * (qy + p.ny * qz);
                    atomicAdd(g + cell, make_float4(wz * fx, wz * fy, wz * fz, 0.f));
                    mark_segment(cell, seg_mask, seg_list, seg_count);
                }
            }
        }
    }
    if (!tiled) return;
    __syncthreads();
    if (by_rows) {
        dilate_rows(binrow, rowmask, T);
        __syncthreads();
    }
    pdl_wait();
    spread_flush(T, tile, by_rows ? rowmask : nullptr, list_all, new_segs, cap, inv_scale, g, seg_mask, seg_list, seg_count, p);
}

// ---------------------------------------------------------------------------------------------
// S2, the two other forms the north_star names ("gather-by-cell over Morton-sorted nodes or
// warp-aggregated atomics, whichever the counters favour"; the paper's own
// fluid3d_force_distribute_kernel is gather-shaped, L356-362).  All nodes with the same base cell
// b = floor(X) - 1 (a "bin") spread into the SAME 4 x 4 x 4 cells.
//   AGGREGATE (warp-aggregated atomics, spread_warp_kernel): a warp takes 32 consecutive nodes, one
//     per lane (along the hidden Morton order they are neighbours on the surface: about 4 share a
//     bin), groups them by bin with match.any, and then serves the groups one after the other:
//     lane = (ox, oy, oz mod 2) owns the two cells (ox, oy, oz) and (ox, oy, oz + 2) of the bin's
//     stencil, reads the group's node records as shared-memory broadcasts, sums W F over the group
//     IN REGISTERS (in lane order: deterministic) and issues one shared-memory atomic per (group,
//     cell, component) instead of one per (node, cell, component).  No block-wide sort, no barrier
//     inside the node loop.
//   GATHER (no atomics at all, spread_gather_kernel): the nodes of a chunk are counting-sorted by bin
//     in shared memory; one thread per tile cell sums W F over the nodes of the (up to) 4 x 4 x 4
//     bins whose stencil contains the cell, and adds the total to its own tile cell.  Each product
//     W F 2^k is rounded to an integer on its own -- by the magic-number addition
//     fma(w, f, 1.5 * 2^23), a full-rate FMA instead of a quarter-rate F2I -- so the result does not
//     depend on the order inside a bin, which the counting sort does not fix.
// Both accumulate into the same 32-bit fixed-point tile as the scatter form.
// ---------------------------------------------------------------------------------------------
constexpr int BIN_CHUNK = IB_THREADS;              // nodes sorted per pass: one per thread
constexpr float FIX_MAGIC = 12582912.0f;           // 1.5 * 2^23
constexpr int FIX_MAGIC_BITS = 0x4B400000;

// direct path of a range whose bounding box does not fit the tile: one RED per (node, cell)
__device__ __forceinline__ void spread_direct(const double* __restrict__ X, const double* __restrict__ Y,
                                              const double* __restrict__ Z, const float4* __restrict__ F, const int n0,
                                              const int n1, float4* __restrict__ g, unsigned* __restrict__ seg_mask,
                                              int* __restrict__ seg_list, int* __restrict__ seg_count, const LbmParams& p) {
    const int sub = threadIdx.x & (SPREAD_LANES - 1), ox = sub & 3, oy = sub >> 2;
    for (int m = n0 + (int)threadIdx.x / SPREAD_LANES; m < n1; m += SPREAD_GROUPS) {
        const double x = X[m], y = Y[m], z = Z[m];
        const float4 Fm = __ldg(F + m);
        const double fx = floor(x), fy = floor(y), fz = floor(z);
        float sx, cx, sy, cy, sz, cz;
        sincospif(0.5f * (float)(x - fx), &sx, &cx);
        sincospif(0.5f * (float)(y - fy), &sy, &cy);
        sincospif(0.5f * (float)(z - fz), &sz, &cz);
        const int qx = wrap_index((int)fx - 1 + ox, p.nx, p.wall[0]), qy = wrap_index((int)fy - 1 + oy, p.ny, p.wall[1]);
        if (qx < 0 || qy < 0) continue;
        const float wxy = weight_o(sx, cx, ox) * weight_o(sy, cy, oy);
        const float gx = wxy * Fm.x, gy = wxy * Fm.y, gz = wxy * Fm.z;
#pragma unroll
        for (int oz = 0; oz < 4; ++oz) {
            const int qz = wrap_index((int)fz - 1 + oz, p.nz, p.wall[2]);
            if (qz < 0) continue;
            const float wz = weight_o(sz, cz, oz);
            const int cell = qx + p.nx * (qy + p.ny * qz);
            atomicAdd(g + cell, make_float4(wz * gx, wz * gy, wz * gz, 0.f));
            mark_segment(cell, seg_mask, seg_list, seg_count);
        }
    }
}

// in-place exclusive prefix sum of a[0 .. n) in shared memory, a[n] = total; all threads call it
__device__ __forceinline__ void block_exclusive_scan(int* __restrict__ a, const int n, int* __restrict__ warp_tot) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int items = (n + IB_THREADS - 1) / IB_THREADS, first = tid * items;
    int sum = 0;
    for (int i = 0; i < items; ++i) sum += first + i < n ? a[first + i] : 0;
    int incl = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
    }
    if (lane == 31) warp_tot[warp] = incl;
    __syncthreads();
    if (warp == 0) {
        const int w = lane < IB_THREADS / 32 ? warp_tot[lane] : 0;
        int wi = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, wi, o);
            if (lane >= o) wi += v;
        }
        if (lane < IB_THREADS / 32) warp_tot[lane] = wi - w;
        if (lane == IB_THREADS / 32 - 1) a[n] = wi;
    }
    __syncthreads();
    int run = warp_tot[warp] + incl - sum;
    for (int i = 0; i < items; ++i)
        if (first + i < n) {
            const int v = a[first + i];
            a[first + i] = run;
            run += v;
        }
    __syncthreads();
}

__global__ void __launch_bounds__(IB_THREADS, 1024 / IB_THREADS) spread_gather_kernel(
    const double* __restrict__ X, const double* __restrict__ Y, const double* __restrict__ Z,
    const float4* __restrict__ F, const int2* __restrict__ ranges, float4* __restrict__ g,
    unsigned* __restrict__ seg_mask, int* __restrict__ seg_list, int* __restrict__ seg_count, const LbmParams p,
    const int cap, int* __restrict__ range_box, const int box_cap, const bool list_all) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ MeshTile T;
    __shared__ int warp_tot[IB_THREADS / 32];
    int* tile = reinterpret_cast<int*>(smem_raw);                      // [3][cap] fixed point, padded pitches
    int* new_segs = tile + 3 * cap;                                    // [SPREAD_SEG_LIST]
    int* bin_start = new_segs + SPREAD_SEG_LIST;                       // [cap + 4] counts, then first slot of each bin
    float4* rec = reinterpret_cast<float4*>(bin_start + ((cap + 4) & ~3));   // [3][BIN_CHUNK] sorted node records
    unsigned* binrow = reinterpret_cast<unsigned*>(rec + 3 * BIN_CHUNK);     // [cap / 4] occupied base cells, x-mask per tile row
    unsigned* rowmask = binrow + cap / 4;                              // [cap / 4] touched cells, x-mask per tile row
    const int2 range = __ldg(ranges + blockIdx.x);
    const int n0 = range.x, n1 = range.y, tid = threadIdx.x;
    tile_setup(T, X, Y, Z, F, n0, n1, p, cap, true, (int)blockIdx.x < box_cap ? range_box + 8 * blockIdx.x : nullptr);
    const float fmax = __uint_as_float(T.fmax_bits);
    if (T.enabled == 0 || !(fmax < 3.0e38f)) {
        pdl_wait();
        spread_direct(X, Y, Z, F, n0, n1, g, seg_mask, seg_list, seg_count, p);
        return;
    }
    // |tile value| <= n_nodes max W max|F| 2^k < 2^30 and every product |W F 2^k| <= max|F| 2^k / 8 < 2^22
    // (a range without force still runs: its cells are listed for the interpolation)
    const int k = fmax > 0.f ? max(-100, min(100, min(29 - ilogbf(0.125f * (float)(n1 - n0) * fmax), 21 - ilogbf(0.125f * fmax)))) : 0;
    const float scale = ldexpf(1.0f, k), inv_scale = ldexpf(1.0f, -k);
    const int p0 = T.p0, pp = T.pp, nword = pp * T.e[2];
    for (int t = tid; t < nword; t += IB_THREADS) {
        tile[t] = 0; tile[cap + t] = 0; tile[2 * cap + t] = 0;
    }
    const bool by_rows = list_all && T.e[0] <= 32;
    if (by_rows)
        for (int t = tid; t < T.e[1] * T.e[2]; t += IB_THREADS) binrow[t] = 0u;
    const int nb0 = T.e[0] - 3, nb1 = T.e[1] - 3, nb2 = T.e[2] - 3, nbins = nb0 * nb1 * nb2;
    const bool clipped = T.clipped != 0;
    const int n_chunks = (n1 - n0 + BIN_CHUNK - 1) / BIN_CHUNK;
    for (int c = 0; c < n_chunks; ++c) {
        const int c0 = n0 + (int)((long)(n1 - n0) * c / n_chunks), c1 = n0 + (int)((long)(n1 - n0) * (c + 1) / n_chunks);
        for (int b = tid; b <= nbins; b += IB_THREADS) bin_start[b] = 0;
        __syncthreads();                                               // also: tile zeroed / previous chunk consumed
        // ---- one node per thread: its bin, its rank inside the bin, its record
        const bool have = c0 + tid < c1;
        int bin = 0, rank = 0;
        float4 r0 = make_float4(0.f, 0.f, 0.f, 0.f), r1 = r0, r2 = r0;
        if (have) {
            const int m = c0 + tid;
            const double x = X[m], y = Y[m], z = Z[m];
            const float4 Fm = __ldg(F + m);
            const double fx = floor(x), fy = floor(y), fz = floor(z);
            const int bx = (int)fx - 1 - T.o[0], by = (int)fy - 1 - T.o[1], bz = (int)fz - 1 - T.o[2];
            bin = (bz * nb1 + by) * nb0 + bx;
            rank = atomicAdd(bin_start + bin, 1);
            sincospif(0.5f * (float)(x - fx), &r0.x, &r0.y);
            sincospif(0.5f * (float)(y - fy), &r0.z, &r0.w);
            sincospif(0.5f * (float)(z - fz), &r1.x, &r1.y);
            r1.z = Fm.x * scale; r1.w = Fm.y * scale; r2.x = Fm.z * scale;
            r2.y = __int_as_float(bx);
            if (by_rows) touch_base(binrow, T, bx, by, bz);             // binrow was zeroed before the barrier above
        }
        __syncthreads();
        block_exclusive_scan(bin_start, nbins, warp_tot);
        if (have) {
            const int slot = bin_start[bin] + rank;
            rec[slot] = r0; rec[BIN_CHUNK + slot] = r1; rec[2 * BIN_CHUNK + slot] = r2;
        }
        __syncthreads();
        {
            // ---- one thread per tile cell: the bins (bx, by, bz) with cell - bin in {0..3}^3; the x-run
            // of bins of one (by, bz) row is one run of sorted nodes
            const int e0 = T.e[0], e1 = T.e[1], ncell = e0 * e1 * T.e[2];
            for (int t = tid; t < ncell; t += IB_THREADS) {
                const int x = t % e0, r = t / e0;
                const int y = r % e1, z = r / e1;
                if (clipped && (x < T.lo[0] || x >= T.hi[0] || y < T.lo[1] || y >= T.hi[1] || z < T.lo[2] || z >= T.hi[2])) continue;
                const int bx_lo = max(0, x - 3), bx_hi = min(nb0 - 1, x);
                int ax_ = 0, ay_ = 0, az_ = 0, n_add = 0;
                for (int bz = max(0, z - 3); bz <= min(nb2 - 1, z); ++bz)
                    for (int by = max(0, y - 3); by <= min(nb1 - 1, y); ++by) {
                        const int row = (bz * nb1 + by) * nb0;
                        const int js = bin_start[row + bx_lo], je = bin_start[row + bx_hi + 1];
                        const int oy = y - by, oz = z - bz;
                        for (int j = js; j < je; ++j) {
                            const float4 q0 = rec[j], q1 = rec[BIN_CHUNK + j], q2 = rec[2 * BIN_CHUNK + j];
                            const int ox = x - __float_as_int(q2.y);
                            const float wxy = weight_o(q0.x, q0.y, ox) * weight_o(q0.z, q0.w, oy);
                            const float wz = weight_o(q1.x, q1.y, oz);
                            ax_ += __float_as_int(fmaf(wz, wxy * q1.z, FIX_MAGIC));
                            ay_ += __float_as_int(fmaf(wz, wxy * q1.w, FIX_MAGIC));
                            az_ += __float_as_int(fmaf(wz, wxy * q2.x, FIX_MAGIC));
                        }
                        n_add += je - js;
                    }
                const int bias = n_add * FIX_MAGIC_BITS, w = z * pp + y * p0 + x;
                tile[w] += ax_ - bias; tile[cap + w] += ay_ - bias; tile[2 * cap + w] += az_ - bias;
            }
        }
        __syncthreads();                                               // bins and records consumed
    }
    if (by_rows) {
        dilate_rows(binrow, rowmask, T);
        __syncthreads();
    }
    pdl_wait();
    spread_flush(T, tile, by_rows ? rowmask : nullptr, list_all, new_segs, cap, inv_scale, g, seg_mask, seg_list, seg_count, p);
}

__global__ void __launch_bounds__(IB_THREADS, 1024 / IB_THREADS) spread_warp_kernel(
    const double* __restrict__ X, const double* __restrict__ Y, const double* __restrict__ Z,
    const float4* __restrict__ F, const int2* __restrict__ ranges, float4* __restrict__ g,
    unsigned* __restrict__ seg_mask, int* __restrict__ seg_list, int* __restrict__ seg_count, const LbmParams p,
    const int cap, int* __restrict__ range_box, const int box_cap, const bool list_all) {
    constexpr unsigned FULL = 0xffffffffu;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ MeshTile T;
    int* tile = reinterpret_cast<int*>(smem_raw);                      // [3][cap] fixed point, padded pitches
    int* new_segs = tile + 3 * cap;                                    // [SPREAD_SEG_LIST]
    float4* rec = reinterpret_cast<float4*>(new_segs + SPREAD_SEG_LIST);   // [warp][3][32] node records
    unsigned* binrow = reinterpret_cast<unsigned*>(rec + 3 * IB_THREADS);    // [cap / 4] occupied base cells, x-mask per tile row
    unsigned* rowmask = binrow + cap / 4;                              // [cap / 4] touched cells, x-mask per tile row
    const int2 range = __ldg(ranges + blockIdx.x);
    const int n0 = range.x, n1 = range.y, tid = threadIdx.x;
    tile_setup(T, X, Y, Z, F, n0, n1, p, cap, true, (int)blockIdx.x < box_cap ? range_box + 8 * blockIdx.x : nullptr);
    const float fmax = __uint_as_float(T.fmax_bits);
    if (T.enabled == 0 || !(fmax < 3.0e38f)) {
        pdl_wait();
        spread_direct(X, Y, Z, F, n0, n1, g, seg_mask, seg_list, seg_count, p);
        return;
    }
    // |tile value| <= n_nodes max W max|F| 2^k < 2^30 (a range without force still runs: its cells are listed)
    const int k = fmax > 0.f ? max(-100, min(100, 29 - ilogbf(0.125f * (float)(n1 - n0) * fmax))) : 0;
    const float scale = ldexpf(1.0f, k), inv_scale = ldexpf(1.0f, -k);
    const int p0 = T.p0, pp = T.pp, nword = pp * T.e[2];
    for (int t = tid; t < nword; t += IB_THREADS) {
        tile[t] = 0; tile[cap + t] = 0; tile[2 * cap + t] = 0;
    }
    const bool by_rows = list_all && T.e[0] <= 32;
    if (by_rows)
        for (int t = tid; t < T.e[1] * T.e[2]; t += IB_THREADS) binrow[t] = 0u;
    const bool clipped = T.clipped != 0;
    __syncthreads();
    const int lane = tid & 31, warp = tid >> 5;
    float4* wrec = rec + warp * 96;
    const int ox = lane & 3, oy = (lane >> 2) & 3, h = lane >> 4;
    const bool xc = ox & 1, yc = oy & 1;                               // this lane's weights use cos (odd offset) or sin
    const float ax = (ox == 0 || ox == 3) ? -0.25f : 0.25f, ay = (oy == 0 || oy == 3) ? -0.25f : 0.25f;
    const float az = h ? 0.25f : -0.25f;     // oz = h: (0: 1/4 - s/4, 1: 1/4 + c/4); oz = h + 2: the opposite sign
    for (int base = n0 + warp * 32; base < n1; base += IB_THREADS) {
        // ---- one node per lane: its record and its bin (tile coordinates of the stencil's first cell, < 1024)
        const int m = base + lane;
        const bool have = m < n1;
        int key = -1;
        if (have) {
            const double x = X[m], y = Y[m], z = Z[m];
            const float4 Fm = __ldg(F + m);
            const double fx = floor(x), fy = floor(y), fz = floor(z);
            key = ((int)fx - 1 - T.o[0]) | (((int)fy - 1 - T.o[1]) << 10) | (((int)fz - 1 - T.o[2]) << 20);
            float4 r0, r1;
            sincospif(0.5f * (float)(x - fx), &r0.x, &r0.y);
            sincospif(0.5f * (float)(y - fy), &r0.z, &r0.w);
            sincospif(0.5f * (float)(z - fz), &r1.x, &r1.y);
            r1.z = Fm.x * scale; r1.w = Fm.y * scale;
            wrec[lane] = r0; wrec[32 + lane] = r1; wrec[64 + lane] = make_float4(Fm.z * scale, 0.f, 0.f, 0.f);
        }
        __syncwarp();
        const unsigned peers = __match_any_sync(FULL, key);
        unsigned todo = __ballot_sync(FULL, have && (__ffs(peers) - 1) == lane);   // the first lane of every group
        while (todo) {
            const int src = __ffs(todo) - 1;
            todo &= todo - 1;
            unsigned members = __shfl_sync(FULL, peers, src);
            const int kk = __shfl_sync(FULL, key, src);
            const int bx = kk & 1023, by = (kk >> 10) & 1023, bz = kk >> 20;
            float a0x = 0.f, a0y = 0.f, a0z = 0.f, a1x = 0.f, a1y = 0.f, a1z = 0.f;
            while (members) {                                          // in lane order: a fixed summation order
                const int j = __ffs(members) - 1;
                members &= members - 1;
                const float4 q0 = wrec[j], q1 = wrec[32 + j];
                const float fzc = wrec[64 + j].x;
                const float wx = fmaf(ax, xc ? q0.y : q0.x, 0.25f);
                const float wy = fmaf(ay, yc ? q0.w : q0.z, 0.25f);
                const float tz = h ? q1.y : q1.x;
                const float wlo = fmaf(az, tz, 0.25f), whi = fmaf(-az, tz, 0.25f);
                const float wxy = wx * wy;
                const float gx = wxy * q1.z, gy = wxy * q1.w, gz = wxy * fzc;
                a0x = fmaf(wlo, gx, a0x); a0y = fmaf(wlo, gy, a0y); a0z = fmaf(wlo, gz, a0z);
                a1x = fmaf(whi, gx, a1x); a1y = fmaf(whi, gy, a1y); a1z = fmaf(whi, gz, a1z);
            }
            const int tx = bx + ox, ty = by + oy, tz0 = bz + h, tz1 = bz + h + 2;
            if (by_rows && lane == src) touch_base(binrow, T, bx, by, bz);
            if (clipped && (tx < T.lo[0] || tx >= T.hi[0] || ty < T.lo[1] || ty >= T.hi[1])) continue;
            const int t0 = tz0 * pp + ty * p0 + tx, t1 = t0 + 2 * pp;
            if (!clipped || (tz0 >= T.lo[2] && tz0 < T.hi[2])) {
                atomicAdd(tile + t0, __float2int_rn(a0x));
                atomicAdd(tile + cap + t0, __float2int_rn(a0y));
                atomicAdd(tile + 2 * cap + t0, __float2int_rn(a0z));
            }
            if (!clipped || (tz1 >= T.lo[2] && tz1 < T.hi[2])) {
                atomicAdd(tile + t1, __float2int_rn(a1x));
                atomicAdd(tile + cap + t1, __float2int_rn(a1y));
                atomicAdd(tile + 2 * cap + t1, __float2int_rn(a1z));
            }
        }
        __syncwarp();                                                  // records consumed
    }
    __syncthreads();
    if (by_rows) {
        dilate_rows(binrow, rowmask, T);
        __syncthreads();
    }
    pdl_wait();
    spread_flush(T, tile, by_rows ? rowmask : nullptr, list_all, new_segs, cap, inv_scale, g, seg_mask, seg_list, seg_count, p);
}

// zero the cells of the segments the previous spread touched (its list), and drop their activity
// bits: 8 lanes per segment, one float4 each = one 128-byte line per segment.  Also resets the
// counter the coming spread will append to (the two counters alternate).
__global__ void __launch_bounds__(256) clear_spread_kernel(float4* __restrict__ g, unsigned* __restrict__ seg_mask,
                                                           const int* __restrict__ seg_list, const int* __restrict__ count_done,
                                                           int* __restrict__ count_next, const int cells) {
    pdl_launch_dependents();                                           // the spread kernel may start its prologue
    const int n = *count_done;
    const int lane8 = threadIdx.x & (SEG - 1);
    const int stride = gridDim.x * (256 / SEG);
    for (int e = blockIdx.x * (256 / SEG) + (threadIdx.x >> SEG_SHIFT); e < n; e += stride) {
        const int seg = __ldg(seg_list + e);
        const int c = seg * SEG + lane8;
        if (c < cells) g[c] = make_float4(0.f, 0.f, 0.f, 0.f);
        if (lane8 == 0) seg_mask[seg >> 5] = 0u;          // every set bit of the word is in the list
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) *count_next = 0;
}

// S4 pre-pass: (vx, vy, vz, rho) of the state after lbm_step for every cell of the 8-cell segments
// the last ib_spread listed -- exactly the cells inside some node's stencil (plus the rounding to
// aligned segments).  Eight adjacent lanes pull the 19 populations of eight adjacent cells: every
// load instruction of the group reads one whole 32-byte sector of a population row, and the result
// is one 128-byte line of the velocity field.  The interpolation kernel then fills its tile from
// that field instead of gathering 19 scattered values per tile cell (whose 12-cell tile rows used
// 2.4 x the sectors they needed).
__global__ void __launch_bounds__(256, 4) segment_macros_kernel(const float* __restrict__ src, const float4* __restrict__ g,
                                                             const int* __restrict__ seg_list, const int* __restrict__ seg_count,
                                                             float4* __restrict__ vfield, const LbmParams p) {
    pdl_launch_dependents();                                           // the listed-cells kernel may stage its positions
    const int n = *seg_count;
    const int lane8 = threadIdx.x & (SEG - 1);
    const int stride = gridDim.x * (256 / SEG);
    for (int e = blockIdx.x * (256 / SEG) + (threadIdx.x >> SEG_SHIFT); e < n; e += stride) {
        const int cell = __ldg(seg_list + e) * SEG + lane8;
        if (cell >= p.cells) continue;
        const Cell c = cell_of(cell, p);
        const bool interior = c.i >= 1 && c.i <= p.nx - 2 && c.j >= 1 && c.j <= p.ny - 2 && c.k >= 1 && c.k <= p.nz - 2;
        vfield[cell] = interior ? cell_macros_interior(src, g, p, cell) : cell_macros(src, g, p, c);
    }
}

// one lane's column of the gather from the shared velocity tile
template <bool CHECK>
__device__ __forceinline__ void gather_column(const float4* __restrict__ tile, const MeshTile& T, const NodeStencil& st,
                                              const int tx, float& ux, float& uy, float& uz) {
    const int e0 = T.e[0], e10 = T.e[0] * T.e[1];
    if (CHECK && (tx < T.lo[0] || tx >= T.hi[0])) return;
    const float4* col = tile + ((st.bz * T.e[1] + st.by) * e0 + tx);
#pragma unroll
    for (int oz = 0; oz < 4; ++oz) {
        if (CHECK && (st.bz + oz < T.lo[2] || st.bz + oz >= T.hi[2])) continue;
#pragma unroll
        for (int oy = 0; oy < 4; ++oy) {
            if (CHECK && (st.by + oy < T.lo[1] || st.by + oy >= T.hi[1])) continue;
            const float W = st.wy[oy] * st.wz[oz];
            const float4 v = col[oz * e10 + oy * e0];
            ux = fmaf(W, v.x, ux);
            uy = fmaf(W, v.y, uy);
            uz = fmaf(W, v.z, uz);
        }
    }
}

// S4 + S5 right after ib_spread for the same positions (the coupled loop).  Every cell of every
// node's stencil is then in a listed segment, so its (v, rho) is in the velocity field
// segment_macros_kernel just wrote, and the bounding box of the range is the one the spread
// stored.  The block copies the box out of the field into its shared-memory tile -- whole rows,
// coalesced, L2 hits; cells of the box that no stencil contains hold older finite values that no
// node reads -- and the nodes gather from the tile.  No bounding-box pass, no marks, no
// compaction, no pull.  The positions of the range are staged in
// shared memory (one coalesced load, in flight while the tile fills), so the gather sweeps run
// without a global-load stall and every read of a position precedes every write.
// A range whose box does not fit the tile (or PLB_INTERP=direct) gathers straight from the field.
constexpr int INTERP_STAGE = 1024;     // positions of the first nodes of a range are staged in shared memory

__device__ __forceinline__ void interpolate_node(double* __restrict__ X, double* __restrict__ Y, double* __restrict__ Z,
                                                 float4* __restrict__ U, const float4* __restrict__ tile,
                                                 const float4* __restrict__ vfield, const MeshTile& T, const bool tiled,
                                                 const double x, const int m, const bool valid, const int sub,
                                                 const int o0, const int o1, const int o2, int* __restrict__ counters,
                                                 const LbmParams& p) {
    const NodeStencil st = node_stencil<true>(x, sub, o0, o1, o2);
    float ux = 0.f, uy = 0.f, uz = 0.f;
    if (!valid) {
    } else if (tiled) {
        if (T.clipped) gather_column<true>(tile, T, st, st.bx + sub, ux, uy, uz);
        else           gather_column<false>(tile, T, st, st.bx + sub, ux, uy, uz);
    } else {
        const int qx = wrap_index(st.bx + sub, p.nx, p.wall[0]);
        if (qx >= 0) {
            int row[4];                                               // qx + nx * qy, or -1
#pragma unroll
            for (int oy = 0; oy < 4; ++oy) {
                const int qy = wrap_index(st.by + oy, p.ny, p.wall[1]);
                row[oy] = qy < 0 ? -1 : qx + p.nx * qy;
            }
            const int sz = p.nx * p.ny;
#pragma unroll
            for (int oz = 0; oz < 4; ++oz) {
                const int qz = wrap_index(st.bz + oz, p.nz, p.wall[2]);
                if (qz < 0) continue;
#pragma unroll
                for (int oy = 0; oy < 4; ++oy) {
                    if (row[oy] < 0) continue;
                    const float W = st.wy[oy] * st.wz[oz];
                    const float4 v = __ldg(vfield + (row[oy] + sz * qz));
                    ux = fmaf(W, v.x, ux);
                    uy = fmaf(W, v.y, uy);
                    uz = fmaf(W, v.z, uz);
                }
            }
        }
    }
    ux *= st.wx; uy *= st.wx; uz *= st.wx;
#pragma unroll
    for (int o = NODE_LANES / 2; o > 0; o >>= 1) {
        ux += __shfl_xor_sync(0xffffffffu, ux, o);
        uy += __shfl_xor_sync(0xffffffffu, uy, o);
        uz += __shfl_xor_sync(0xffffffffu, uz, o);
    }
    // the lane of axis a advances coordinate a (it holds the old value: no second read)
    const float ua = sub == 1 ? uy : (sub == 2 ? uz : ux);
    if (valid && sub < 3) {
        const double xn = x + (double)ua;
        (sub == 1 ? Y : (sub == 2 ? Z : X))[m] = xn;
        // halfway bounce-back walls lie at -1/2 and n - 1/2, on-site velocity walls at 0 and n - 1
        const int na = sub == 1 ? p.ny : (sub == 2 ? p.nz : p.nx);
        const double ma = p.wall[sub] == PLB_WALL_HH ? 0.0 : 0.5;
        if (p.wall[sub] && (xn < -ma || xn > (double)(na - 1) + ma)) atomicOr(counters + 1, STATUS_NODE_LEFT);
    }
    if (valid && sub == 3) U[m] = make_float4(ux, uy, uz, 0.f);
}

__global__ void __launch_bounds__(IB_THREADS, 1024 / IB_THREADS) interpolate_listed_kernel(
    double* __restrict__ X, double* __restrict__ Y, double* __restrict__ Z, float4* __restrict__ U,
    const int2* __restrict__ ranges, const float4* __restrict__ vfield, const int* __restrict__ range_box,
    const int box_cap, int* __restrict__ counters, const LbmParams p, const int cap, const bool use_tile) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ MeshTile T;
    float4* tile = reinterpret_cast<float4*>(smem_raw);                // [cap] (vx, vy, vz, rho)
    const int2 range = __ldg(ranges + blockIdx.x);
    const int n0 = range.x, n1 = range.y, tid = threadIdx.x;
    const int sub = tid & (NODE_LANES - 1), group = tid / NODE_LANES;
    double* pos = reinterpret_cast<double*>(tile + cap);               // [3][INTERP_STAGE]
    const int n_staged = min(n1 - n0, INTERP_STAGE);
    for (int i = tid; i < n_staged; i += IB_THREADS) {
        pos[i] = X[n0 + i]; pos[INTERP_STAGE + i] = Y[n0 + i]; pos[2 * INTERP_STAGE + i] = Z[n0 + i];
    }
    if (!use_tile) {
        if (tid == 0) T.enabled = 0;
        __syncthreads();
    } else if ((int)blockIdx.x < box_cap) {
        if (tid == 0) {
            const int4 b0 = __ldg(reinterpret_cast<const int4*>(range_box) + 2 * blockIdx.x);
            const int4 b1 = __ldg(reinterpret_cast<const int4*>(range_box) + 2 * blockIdx.x + 1);
            T.mn[0] = b0.x; T.mn[1] = b0.y; T.mn[2] = b0.z;
            T.mx[0] = b1.x; T.mx[1] = b1.y; T.mx[2] = b1.z;
            tile_geometry(T, b0.w != 0, p, cap, false);
        }
        __syncthreads();
    } else {
        tile_setup(T, X, Y, Z, nullptr, n0, n1, p, cap, false);
    }
    const bool tiled = T.enabled != 0;
    const int o0 = tiled ? T.o[0] : 0, o1 = tiled ? T.o[1] : 0, o2 = tiled ? T.o[2] : 0;
    pdl_wait();                                                        // the pre-pass has written the velocity field
    if (tiled) {
        const int e0 = T.e[0], e1 = T.e[1], ncell = e0 * e1 * T.e[2];
        const TileSplit split(T);
        if (T.interior) {
            const int sy = p.nx, sz = p.nx * p.ny;
            const int origin = T.o[0] + sy * T.o[1] + sz * T.o[2];
            for (int t = tid; t < ncell; t += IB_THREADS) {
                int x, y, z;
                split(t, x, y, z);
                tile[t] = __ldg(vfield + (origin + x + sy * y + sz * z));
            }
        } else {
            for (int t = tid; t < ncell; t += IB_THREADS) {
                int x, y, z;
                split(t, x, y, z);
                if (x < T.lo[0] || x >= T.hi[0] || y < T.lo[1] || y >= T.hi[1] || z < T.lo[2] || z >= T.hi[2]) continue;
                const Cell c = tile_cell(T, x, y, z, p);
                tile[t] = __ldg(vfield + (c.i + p.nx * (c.j + p.ny * c.k)));
            }
        }
    }
    __syncthreads();                                                   // positions staged (and the tile filled)
    for (int mb = n0; mb < n1; mb += IB_GROUPS) {
        const int m = mb + group;
        const bool valid = m < n1;
        double x = 0.0;                                                // (lanes without a node only run the shuffles)
        if (valid) x = m - n0 < INTERP_STAGE ? pos[min(sub, 2) * INTERP_STAGE + (m - n0)] : node_coord(X, Y, Z, m, sub);
        interpolate_node(X, Y, Z, U, tile, vfield, T, tiled, x, m, valid, sub, o0, o1, o2, counters, p);
    }
}

// S4 + S5, PULL form: no velocity field at all.  The block finds the tile cells some node of its
// range needs (one bit per node for its base cell, dilated by the 4 x 4 x 4 stencil: the marks of
// the spread), compacts them, computes their (v, rho) straight from the 19 populations each cell
// pulls out of the post-collision lattice, and gathers.  Sparsely sampled meshes (config 4: a tile
// cell is needed by one mesh only) take this form: the pull of one block overlaps the gather of
// another on the same SM, which a bandwidth-bound pre-pass followed by a latency-bound gather
// kernel cannot (config 4: 0.16 ms against 0.19 ms; at config 5, where a cell lies in ~14 tiles,
// the pre-pass computes it once and wins: 1.33 against 1.51 ms).  It also serves every call order
// (passive advection, moved nodes): the box of the range comes from the last spread only when that
// spread saw these positions, else from a pass over the positions.
__global__ void __launch_bounds__(IB_THREADS, 1024 / IB_THREADS) interpolate_pull_kernel(
    double* __restrict__ X, double* __restrict__ Y, double* __restrict__ Z, float4* __restrict__ U,
    const int2* __restrict__ ranges, const float* __restrict__ src, const float4* __restrict__ g,
    const int* __restrict__ range_box, const int box_cap, int* __restrict__ counters, const LbmParams p,
    const int cap) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ MeshTile T;
    float4* tile = reinterpret_cast<float4*>(smem_raw);                // [cap] (vx, vy, vz, rho)
    unsigned short* list = reinterpret_cast<unsigned short*>(tile + cap);   // [cap] needed tile cells
    const int2 range = __ldg(ranges + blockIdx.x);
    const int n0 = range.x, n1 = range.y, tid = threadIdx.x;
    const int sub = tid & (NODE_LANES - 1), group = tid / NODE_LANES;
    // (no staging of the positions in shared memory: the pull below wants the L1 cache that
    // shared memory takes away -- 24 KB more per block cost 40 % of the kernel, measured twice)
    if ((int)blockIdx.x < box_cap) {
        if (tid == 0) {
            const int4 b0 = __ldg(reinterpret_cast<const int4*>(range_box) + 2 * blockIdx.x);
            const int4 b1 = __ldg(reinterpret_cast<const int4*>(range_box) + 2 * blockIdx.x + 1);
            T.mn[0] = b0.x; T.mn[1] = b0.y; T.mn[2] = b0.z;
            T.mx[0] = b1.x; T.mx[1] = b1.y; T.mx[2] = b1.z;
            T.n_need = 0;
            tile_geometry(T, b0.w != 0, p, cap, 0);
        }
        __syncthreads();
    } else {
        tile_setup(T, X, Y, Z, nullptr, n0, n1, p, cap, 0);
    }
    const bool tiled = T.enabled != 0;
    const int e0 = T.e[0], e1 = T.e[1], ncell = tiled ? e0 * e1 * T.e[2] : 0;
    const int o0 = tiled ? T.o[0] : 0, o1 = tiled ? T.o[1] : 0, o2 = tiled ? T.o[2] : 0;
    if (tiled) {
        unsigned* binrow = reinterpret_cast<unsigned*>(smem_raw);     // marks alias the (not yet filled) tile
        unsigned* rowmask = binrow + e1 * T.e[2];
        // A densely sampled tile needs all of its cells; so does one wider than a 32-bit row mask.
        const bool by_rows = 2L * (n1 - n0) < (long)ncell && e0 <= 32;
        if (by_rows) {
            for (int t = tid; t < e1 * T.e[2]; t += IB_THREADS) binrow[t] = 0u;
            __syncthreads();
            for (int m = n0 + tid; m < n1; m += IB_THREADS)
                touch_base(binrow, T, (int)floor(X[m]) - 1 - o0, (int)floor(Y[m]) - 1 - o1, (int)floor(Z[m]) - 1 - o2);
            __syncthreads();
            dilate_rows(binrow, rowmask, T);
        }
        __syncthreads();
        // compact the needed cells so that every lane of the moment pass has a cell
        const TileSplit split(T);
        for (int t0 = 0; t0 < ncell; t0 += IB_THREADS) {
            const int t = t0 + tid;
            bool want = false;
            if (t < ncell) {
                int x, y, z;
                split(t, x, y, z);
                if (by_rows) want = ((rowmask[z * e1 + y] >> x) & 1u) != 0u;
                else want = x >= T.lo[0] && x < T.hi[0] && y >= T.lo[1] && y < T.hi[1] && z >= T.lo[2] && z < T.hi[2];
            }
            const unsigned vote = __ballot_sync(0xffffffffu, want);
            int base = 0;
            if ((tid & 31) == 0 && vote) base = atomicAdd(&T.n_need, __popc(vote));
            base = __shfl_sync(0xffffffffu, base, 0);
            if (want) list[base + __popc(vote & ((1u << (tid & 31)) - 1u))] = (unsigned short)t;
        }
        __syncthreads();                                               // the marks are consumed: the tile may be written
        const int n_need = T.n_need;
        if (T.interior) {
            const int sy = p.nx, sz = p.nx * p.ny;
            const int origin = T.o[0] + sy * T.o[1] + sz * T.o[2];
            for (int e = tid; e < n_need; e += IB_THREADS) {
                const int t = list[e];
                int x, y, z;
                split(t, x, y, z);
                tile[t] = cell_macros_interior(src, g, p, origin + x + sy * y + sz * z);
            }
        } else {
            for (int e = tid; e < n_need; e += IB_THREADS) {
                const int t = list[e];
                int x, y, z;
                split(t, x, y, z);
                tile[t] = cell_macros(src, g, p, tile_cell(T, x, y, z, p));
            }
        }
    }
    __syncthreads();                                                   // tile filled
    for (int mb = n0; mb < n1; mb += IB_GROUPS) {
        const int m = mb + group;
        const bool valid = m < n1;
        const int axis = sub < 3 ? sub : 0;
        double x = 0.0;                                                // (lanes without a node only run the shuffles)
        if (valid) x = node_coord(X, Y, Z, m, axis);
        const NodeStencil st = node_stencil<true>(x, sub, o0, o1, o2);
        float ux = 0.f, uy = 0.f, uz = 0.f;
        if (!valid) {
        } else if (tiled) {
            if (T.clipped) gather_column<true>(tile, T, st, st.bx + sub, ux, uy, uz);
            else           gather_column<false>(tile, T, st, st.bx + sub, ux, uy, uz);
        } else {
            const int qx = wrap_index(st.bx + sub, p.nx, p.wall[0]);
            if (qx >= 0) {
#pragma unroll
                for (int oz = 0; oz < 4; ++oz) {
                    const int qz = wrap_index(st.bz + oz, p.nz, p.wall[2]);
                    if (qz < 0) continue;
#pragma unroll
                    for (int oy = 0; oy < 4; ++oy) {
                        const int qy = wrap_index(st.by + oy, p.ny, p.wall[1]);
                        if (qy < 0) continue;
                        const float W = st.wy[oy] * st.wz[oz];
                        Cell c;
                        c.i = qx; c.j = qy; c.k = qz;
                        const float4 v = cell_macros(src, g, p, c);
                        ux = fmaf(W, v.x, ux);
                        uy = fmaf(W, v.y, uy);
                        uz = fmaf(W, v.z, uz);
                    }
                }
            }
        }
        ux *= st.wx; uy *= st.wx; uz *= st.wx;
#pragma unroll
        for (int o = NODE_LANES / 2; o > 0; o >>= 1) {
            ux += __shfl_xor_sync(0xffffffffu, ux, o);
            uy += __shfl_xor_sync(0xffffffffu, uy, o);
            uz += __shfl_xor_sync(0xffffffffu, uz, o);
        }
        // the lane of axis a advances coordinate a (it holds the old value: no second read, and a
        // position is read by its own group only)
        const float ua = sub == 1 ? uy : (sub == 2 ? uz : ux);
        if (valid && sub < 3) {
            const double xn = x + (double)ua;
            (sub == 1 ? Y : (sub == 2 ? Z : X))[m] = xn;
            // halfway bounce-back walls lie at -1/2 and n - 1/2, on-site velocity walls at 0 and n - 1
            const int na = sub == 1 ? p.ny : (sub == 2 ? p.nz : p.nx);
            const double ma = p.wall[sub] == PLB_WALL_HH ? 0.0 : 0.5;
            if (p.wall[sub] && (xn < -ma || xn > (double)(na - 1) + ma)) atomicOr(counters + 1, STATUS_NODE_LEFT);
        }
        if (valid && sub == 3) U[m] = make_float4(ux, uy, uz, 0.f);
    }
}

// positions: device SoA <-> AoS staging buffer (so host transfers are one contiguous copy)
// (also stored order <-> caller's order)
__global__ void __launch_bounds__(256) nodes_transpose_kernel(double* __restrict__ X, double* __restrict__ Y,
                                                              double* __restrict__ Z, double* __restrict__ aos,
                                                              const int* __restrict__ orig, const long n, const bool to_aos) {
    const long t = blockIdx.x * 256L + threadIdx.x;
    if (t >= 3 * n) return;
    const long m = t / 3;
    const int d = (int)(t - 3 * m);
    double* comp = d == 0 ? X : (d == 1 ? Y : Z);
    const long a = 3L * __ldg(orig + m) + d;
    if (to_aos) aos[a] = comp[m];
    else        comp[m] = aos[a];
}

__global__ void philox_kernel(const long n, const uint4* __restrict__ ctr, const uint2* __restrict__ key,
                              uint4* __restrict__ out) {
    const long t = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (t < n) out[t] = philox4x32_10(ctr[t], key[t]);
}

// ---------------------------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------------------------
int launch_membrane_forces(Ctx* c, float sigma, unsigned long long seed, unsigned long long step) {
    if (c->n_nodes == 0) return PLB_OK;
    for (const SpringGroup& grp : c->groups) {                        // one launch per topology group
        const long n = (long)grp.n_meshes * grp.nn;
        node_force_kernel<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(
            c->X[0], c->X[1], c->X[2], c->orig, c->csr_off, c->csr_ent, c->F, grp, sigma, seed, (unsigned)step, c->counters);
        c->launches++;
    }
    if (c->n_cons) {
        constraint_force_kernel<<<(unsigned)c->n_cons, CON_THREADS, 0, c->stream>>>(
            c->X[0], c->X[1], c->X[2], c->tris, c->tri_S0, c->cons, c->F);
        c->launches++;
    }
    const int rc = launch_adhesion_forces(c);
    if (rc) return rc;
    return cuda_check(cudaGetLastError(), "membrane force kernels");
}

// counters[2 + parity] = number of segments listed by the spread of that parity
int launch_clear_spread(Ctx* c, float4* g) {
    const int done = c->list_parity, next = done ^ 1;
    const long want = (c->n_segs + 31) / 32;
    const unsigned grid = (unsigned)(want < (long)c->sm_count * 8 ? (want > 0 ? want : 1) : (long)c->sm_count * 8);
    clear_spread_kernel<<<grid, 256, 0, c->stream>>>(g, c->seg_mask, c->seg_list, c->counters + 2 + done,
                                                     c->counters + 2 + next, c->prm.cells);
    c->list_parity = next;
    c->launches++;
    return cuda_check(cudaGetLastError(), "clear_spread_kernel");
}

static size_t spread_smem(int cap) { return (size_t)cap * 14 + (size_t)SPREAD_SEG_LIST * 4 + (size_t)SPREAD_CHUNK * 48; }
static size_t warp_smem(int cap) { return (size_t)cap * 14 + (size_t)SPREAD_SEG_LIST * 4 + (size_t)IB_THREADS * 48; }
static size_t binned_smem(int cap) {
    return (size_t)cap * 14 + (size_t)SPREAD_SEG_LIST * 4 + (size_t)((cap + 4) & ~3) * 4 + (size_t)BIN_CHUNK * 48;
}
static size_t interp_smem(int cap) { return (size_t)cap * 16 + (((size_t)cap * 2 + 15) & ~(size_t)15); }

// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) once per kernel and size, not once per step
template <typename K>
static int ensure_smem(K kernel, size_t smem, size_t& granted, const char* what) {
    if (smem <= granted) return PLB_OK;
    const int rc = cuda_check(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem), what);
    if (!rc) granted = smem;
    return rc;
}

// Largest tile (in cells) both kernels can hold with at least one block per SM; a tile cell index
// must also fit the 16-bit entries of the interpolation's compact list.
int ib_max_tile_cap() {
    const size_t budget = 200 * 1024;
    const size_t cap = (budget - 64) / 18;
    return (int)(cap < 65535 ? cap : 65535);
}

// words per component of the padded spread tile: two blocks of 113 KB per SM (14 B per word + 20 KB)
int ib_max_spread_cap() { return 6656; }

// Which form of the spread runs: the caller's choice (ib_set_spread_mode), else by how densely the
// tiles are sampled -- measured on the B200 (profiles/r02p_*): the scatter form
// wins on sparsely sampled tiles (config 4: 0.26 nodes per tile cell; 0.098 ms against 0.19 ms), the
// warp-aggregated form on densely sampled ones (config 5: 0.9 per tile cell, about 4 nodes per
// warp-group; 1.38 ms against 1.68 ms).
int spread_mode_of(const Ctx* c) {
    if (c->spread_mode != PLB_SPREAD_AUTO) return c->spread_mode;
    return c->tile_density >= 0.6 ? PLB_SPREAD_AGGREGATE : PLB_SPREAD_SCATTER;
}

// Which form of the interpolation the coupled loop takes: by how densely the tiles are sampled --
// measured on the B200: the pull form on sparsely sampled tiles (config 4: 0.154 ms
// against 0.191 ms), the pre-pass + listed-cells kernel on densely sampled ones, where a cell lies in
// many tiles (config 5: 1.33 ms against 1.52 ms).  PLB_INTERP = "pull" / "tile" / "direct" overrides
// (measurement knob; "direct" = the listed-cells kernel gathering straight from the field).
int interp_form_of(const Ctx* c) {
    if (c->interp_form != PLB_INTERP_AUTO) return c->interp_form;
    return c->tile_density >= 0.6 ? PLB_INTERP_TILE : PLB_INTERP_PULL;
}

// launch with the programmatic-stream-serialization attribute: the kernel may start before the
// preceding kernel of the stream has completed and synchronises with it by griddepcontrol.wait
template <typename... KArgs, typename... Args>
static void launch_overlapped(void (*kernel)(KArgs...), const unsigned grid, const unsigned block, const size_t smem,
                              cudaStream_t stream, const bool overlap, Args... args) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(block); cfg.dynamicSmemBytes = smem; cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = overlap ? 1 : 0;
    cfg.attrs = attr; cfg.numAttrs = 1;
    cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

int launch_spread(Ctx* c, float4* g, bool after_clear) {
    if (c->n_nodes == 0) return PLB_OK;
    static size_t granted_scatter = 0, granted_aggregate = 0, granted_gather = 0;
    const int cap = (c->spread_cap + 3) & ~3;
    int* seg_count = c->counters + 2 + c->list_parity;
    const int mode = spread_mode_of(c);
    // the listed-cells interpolation relies on the list covering every stencil cell
    const bool list_all = interp_form_of(c) != PLB_INTERP_PULL;
    c->listed_all = list_all;
    int rc;
    if (mode == PLB_SPREAD_SCATTER) {
        const size_t smem = spread_smem(cap);
        rc = ensure_smem(spread_mesh_kernel, smem, granted_scatter, "cudaFuncSetAttribute(spread_mesh_kernel)");
        if (rc) return rc;
        launch_overlapped(spread_mesh_kernel, (unsigned)c->n_ranges, IB_THREADS, smem, c->stream, after_clear,
                          c->X[0], c->X[1], c->X[2], c->F, c->ranges, g, c->seg_mask, c->seg_list, seg_count, c->prm, cap, c->range_box, c->box_cap, list_all);
    } else if (mode == PLB_SPREAD_AGGREGATE) {
        const size_t smem = warp_smem(cap);
        rc = ensure_smem(spread_warp_kernel, smem, granted_aggregate, "cudaFuncSetAttribute(spread_warp_kernel)");
        if (rc) return rc;
        launch_overlapped(spread_warp_kernel, (unsigned)c->n_ranges, IB_THREADS, smem, c->stream, after_clear,
                          c->X[0], c->X[1], c->X[2], c->F, c->ranges, g, c->seg_mask, c->seg_list, seg_count, c->prm, cap, c->range_box, c->box_cap, list_all);
    } else {
        const size_t smem = binned_smem(cap);
        rc = ensure_smem(spread_gather_kernel, smem, granted_gather, "cudaFuncSetAttribute(spread_gather_kernel)");
        if (rc) return rc;
        launch_overlapped(spread_gather_kernel, (unsigned)c->n_ranges, IB_THREADS, smem, c->stream, after_clear,
                          c->X[0], c->X[1], c->X[2], c->F, c->ranges, g, c->seg_mask, c->seg_list, seg_count, c->prm, cap, c->range_box, c->box_cap, list_all);
    }
    c->launches++;
    return cuda_check(cudaGetLastError(), "spread kernel");
}

int launch_interpolate_advance(Ctx* c) {
    if (c->n_nodes == 0) return PLB_OK;
    const float4* g = (c->g_last_mode == FORCE_NONE) ? nullptr : c->g_last;
    const int form = interp_form_of(c);
    // Densely sampled meshes, right after an ib_spread that saw these positions and listed every
    // stencil cell: the velocity of the listed segments once (pre-pass), then the listed-cells kernel.
    if (form != PLB_INTERP_PULL && c->spread_current && c->listed_all) {
        const long want = (c->n_segs + 31) / 32;
        const unsigned grid = (unsigned)(want < (long)c->sm_count * 16 ? (want > 0 ? want : 1) : (long)c->sm_count * 16);
        segment_macros_kernel<<<grid, 256, 0, c->stream>>>(c->f[c->cur], g, c->seg_list, c->counters + 2 + c->list_parity,
                                                           c->vfield, c->prm);
        c->launches++;
        static size_t granted_listed = 0;
        const size_t smem_l = (size_t)c->tile_cap * 16 + (size_t)3 * INTERP_STAGE * sizeof(double);
        const int rc = ensure_smem(interpolate_listed_kernel, smem_l, granted_listed, "cudaFuncSetAttribute(interpolate_listed_kernel)");
        if (rc) return rc;
        // a programmatic dependent launch behind the pre-pass: box, geometry and the staging of the
        // positions overlap it, the kernel waits just ahead of its first read of the field
        launch_overlapped(interpolate_listed_kernel, (unsigned)c->n_ranges, IB_THREADS, smem_l, c->stream, true,
                          c->X[0], c->X[1], c->X[2], c->U, c->ranges, c->vfield, c->range_box, c->box_cap, c->counters, c->prm,
                          c->tile_cap, form != PLB_INTERP_DIRECT);
        c->launches++;
        return cuda_check(cudaGetLastError(), "interpolate_listed_kernel");
    }
    // Sparsely sampled meshes, and every other call order (passive advection, moved nodes): the
    // pull form, which needs neither list nor field.
    static size_t granted_pull = 0;
    const size_t smem_p = interp_smem(c->tile_cap);
    const int rc = ensure_smem(interpolate_pull_kernel, smem_p, granted_pull, "cudaFuncSetAttribute(interpolate_pull_kernel)");
    if (rc) return rc;
    interpolate_pull_kernel<<<(unsigned)c->n_ranges, IB_THREADS, smem_p, c->stream>>>(
        c->X[0], c->X[1], c->X[2], c->U, c->ranges, c->f[c->cur], g, c->range_box, c->spread_current ? c->box_cap : 0,
        c->counters, c->prm, c->tile_cap);
    c->launches++;
    return cuda_check(cudaGetLastError(), "interpolate_pull_kernel");
}

int launch_nodes_transpose(Ctx* c, bool to_aos) {
    if (c->n_nodes == 0) return PLB_OK;
    nodes_transpose_kernel<<<(unsigned)((3 * c->n_nodes + 255) / 256), 256, 0, c->stream>>>(
        c->X[0], c->X[1], c->X[2], c->stage, c->orig, c->n_nodes, to_aos);
    c->launches++;
    return cuda_check(cudaGetLastError(), "nodes_transpose_kernel");
}

int launch_philox(cudaStream_t s, long n, const unsigned* ctr, const unsigned* key, unsigned* out) {
    if (n <= 0) return PLB_OK;
    philox_kernel<<<(unsigned)((n + 127) / 128), 128, 0, s>>>(n, (const uint4*)ctr, (const uint2*)key, (uint4*)out);
    return cuda_check(cudaGetLastError(), "philox_kernel");
}

}  // namespace plb
