// ib.cu -- immersed-boundary and membrane kernels (Eq. 2-3, section 3.4.2 Eq. 31-36).
//
// Node data: positions SoA fp64 (unwrapped), forces / node velocities float4 AoS.
// The forcing field is float4 per cell so that the spread is one 128-bit vector atomic per
// (node, cell) pair (red.global.add.v4.f32, sm_90+).
#include <climits>
#include "plb_internal.cuh"
#include "lbm_device.cuh"

namespace plb {

// ---------------------------------------------------------------------------------------------
// S1: per-edge Hookean spring force (Eq. 2-3): e = k (|R| - L) R/|R| on node a, -e on node b.
// R and |R| - L are formed in fp64 (positions reach ~1e3, lengths ~1, stretches ~1e-3), the
// rest in fp32; two vector atomics per edge.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) force_init_kernel(float4* __restrict__ F, const long n, const float sigma,
                                                         const unsigned long long seed, const unsigned step) {
    const long m = blockIdx.x * 256L + threadIdx.x;
    if (m >= n) return;
    float4 f = make_float4(0.f, 0.f, 0.f, 0.f);
    if (sigma > 0.f) {
        // Box-Muller on the four uniforms of counter (node, step, tag 2)
        const uint4 r = noise_words(seed, (unsigned long long)m, step, 2u);
        const float r0 = sqrtf(-2.0f * logf(uniform01(r.x)));
        const float r2 = sqrtf(-2.0f * logf(uniform01(r.z)));
        float s1, c1;
        sincospif(2.0f * uniform01(r.y), &s1, &c1);
        f.x = sigma * r0 * c1;
        f.y = sigma * r0 * s1;
        f.z = sigma * r2 * cospif(2.0f * uniform01(r.w));
    }
    F[m] = f;
}

__global__ void __launch_bounds__(256) edge_force_kernel(const double* __restrict__ X, const double* __restrict__ Y,
                                                         const double* __restrict__ Z, const int2* __restrict__ edges,
                                                         const float2* __restrict__ prm, float4* __restrict__ F,
                                                         const long n_edges, int* __restrict__ counters) {
    const long e = blockIdx.x * 256L + threadIdx.x;
    if (e >= n_edges) return;
    const int2 ab = __ldg(edges + e);
    const float2 Lk = __ldg(prm + e);
    const double rx = __ldg(X + ab.y) - __ldg(X + ab.x);
    const double ry = __ldg(Y + ab.y) - __ldg(Y + ab.x);
    const double rz = __ldg(Z + ab.y) - __ldg(Z + ab.x);
    const double l = sqrt(rx * rx + ry * ry + rz * rz);
    if (!(l > 0.0)) {
        atomicOr(counters + 1, STATUS_ZERO_EDGE);
        return;
    }
    const float s = Lk.y * (float)((l - (double)Lk.x) / l);
    const float ex = s * (float)rx, ey = s * (float)ry, ez = s * (float)rz;
    atomicAdd(F + ab.x, make_float4(ex, ey, ez, 0.f));
    atomicAdd(F + ab.y, make_float4(-ex, -ey, -ez, 0.f));
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
struct Axis {
    int base;      // floor(X) - 1 (unwrapped)
    float s, c;
};

__device__ __forceinline__ Axis axis_of(const double x) {
    const double fl = floor(x);
    Axis a;
    a.base = (int)fl - 1;
    sincospif(0.5f * (float)(x - fl), &a.s, &a.c);
    return a;
}
__device__ __forceinline__ float weight_of(const Axis& a, const int o) {
    const float t = (o == 0) ? -a.s : (o == 1) ? a.c : (o == 2) ? a.s : -a.c;
    return 0.25f + 0.25f * t;
}
// wrapped index on a periodic axis; -1 if dropped on a wall axis
__device__ __forceinline__ int wrap_index(int q, const int n, const int wall) {
    if (q >= 0 && q < n) return q;
    if (wall) return -1;
    q %= n;
    return q < 0 ? q + n : q;
}

// ---------------------------------------------------------------------------------------------
// S2 and S4/S5 run one thread block per NODE RANGE (a mesh, or a slice of a very large mesh).
// A platelet is a compact object: the 4x4x4 supports of its nodes overlap heavily (about 13
// contributions per touched cell at config 4, 1000 at config 5), so the block accumulates /
// gathers through a TILE of the lattice held in shared memory -- the bounding box of the
// supports of its nodes -- and touches global memory once per tile cell:
//   spread:       zero tile -> nodes scatter into the tile -> the non-zero tile cells go to the
//                 forcing field with one 128-bit RED each.  The tile accumulates in 32-bit fixed
//                 point with a per-block power-of-two scale (native shared-memory integer
//                 atomics; the fp32 ones are compare-and-swap loops): order-independent, and
//                 with a resolution of n_nodes/8 * 2^-30 of the largest nodal force component;
//   interpolate:  mark the tile cells some node needs -> compact them -> their v straight from
//                 the 19 pulled populations (no velocity field in HBM) -> nodes gather from the tile.
// A range whose bounding box does not fit the tile (a non-compact "mesh") takes the direct path:
// global REDs per (node, cell) and on-the-fly cell moments.  Both paths compute the same sums.
// Within a block 16 lanes serve one node: lane = (ox, oy), loop over oz.
// ---------------------------------------------------------------------------------------------
constexpr int IB_THREADS = 512;
constexpr int IB_CHUNK = 256;                      // nodes whose stencil records are staged at a time
constexpr int LANES_PER_NODE = 16;
constexpr int IB_GROUPS = IB_THREADS / LANES_PER_NODE;

struct MeshTile {
    int o[3];            // unwrapped lattice coordinate of tile cell (0,0,0)
    int e[3];            // extent in cells
    int lo[3], hi[3];    // tile coordinates [lo, hi) that exist on the lattice (wall axes clip)
    int enabled;
    int mn[3], mx[3];    // reduction scratch: min / max of floor(X)
    unsigned fmax_bits;  // reduction scratch: largest |F| component (non-negative float bits)
    int n_need;          // interpolate: number of tile cells some node needs
};

// set the activity bit of the 8-cell segment of a cell
__device__ __forceinline__ void mark_segment(const int cell, unsigned* __restrict__ seg_mask) {
    const int seg = cell >> SEG_SHIFT;
    const unsigned bit = 1u << (seg & 31);
    unsigned* word = seg_mask + (seg >> 5);
    if ((*(volatile unsigned*)word & bit) == 0u) atomicOr(word, bit);
}

// bounding box of the supports of nodes [n0, n1) -> tile geometry (all threads of the block);
// with F != nullptr also the largest force component of the range
__device__ __forceinline__ void tile_setup(MeshTile& T, const double* __restrict__ X, const double* __restrict__ Y,
                                           const double* __restrict__ Z, const float4* __restrict__ F, const int n0,
                                           const int n1, const LbmParams& p, const int cap) {
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
        const int n[3] = {p.nx, p.ny, p.nz};
        long long vol = 1;
        bool ok = n1 > n0;
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
        }
        T.enabled = ok ? 1 : 0;
    }
    __syncthreads();
}

// global lattice cell of tile cell t (only called for cells inside [lo, hi) on wall axes)
__device__ __forceinline__ Cell tile_cell(const MeshTile& T, const int t, const LbmParams& p) {
    const int x = t % T.e[0], r = t / T.e[0];
    const int y = r % T.e[1], z = r / T.e[1];
    Cell c;
    c.i = wrap_index(T.o[0] + x, p.nx, 0);
    c.j = wrap_index(T.o[1] + y, p.ny, 0);
    c.k = wrap_index(T.o[2] + z, p.nz, 0);
    return c;
}

// per-node stencil records of one chunk of nodes, in shared memory
struct Chunk {
    int* b;        // [3][IB_CHUNK] base = floor(X) - 1, tile-relative if the tile is enabled
    float* sc;     // [6][IB_CHUNK] sin / cos of pi frac / 2 per axis
};

__device__ __forceinline__ void chunk_record(const Chunk& ch, const MeshTile& T, const bool tiled, const int r,
                                             const double x, const double y, const double z) {
    const Axis ax = axis_of(x), ay = axis_of(y), az = axis_of(z);
    ch.b[r] = tiled ? ax.base - T.o[0] : ax.base;
    ch.b[IB_CHUNK + r] = tiled ? ay.base - T.o[1] : ay.base;
    ch.b[2 * IB_CHUNK + r] = tiled ? az.base - T.o[2] : az.base;
    ch.sc[r] = ax.s; ch.sc[IB_CHUNK + r] = ax.c;
    ch.sc[2 * IB_CHUNK + r] = ay.s; ch.sc[3 * IB_CHUNK + r] = ay.c;
    ch.sc[4 * IB_CHUNK + r] = az.s; ch.sc[5 * IB_CHUNK + r] = az.c;
}
__device__ __forceinline__ Axis chunk_axis(const Chunk& ch, const int a, const int r) {
    Axis ax;
    ax.base = ch.b[a * IB_CHUNK + r];
    ax.s = ch.sc[2 * a * IB_CHUNK + r];
    ax.c = ch.sc[(2 * a + 1) * IB_CHUNK + r];
    return ax;
}

// S2: g_ijk += F_m phi phi phi (Eq. 34).  Also sets the activity bits of the touched segments.
__global__ void __launch_bounds__(IB_THREADS) spread_mesh_kernel(
    const double* __restrict__ X, const double* __restrict__ Y, const double* __restrict__ Z,
    const float4* __restrict__ F, const int2* __restrict__ ranges, float4* __restrict__ g,
    unsigned* __restrict__ seg_mask, const LbmParams p, const int cap) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ MeshTile T;
    int* tile = reinterpret_cast<int*>(smem_raw);                      // [3][cap] fixed point
    Chunk ch;
    ch.b = tile + 3 * (size_t)cap;
    ch.sc = reinterpret_cast<float*>(ch.b + 3 * IB_CHUNK);
    float* rF = ch.sc + 6 * IB_CHUNK;                                  // [3][IB_CHUNK]
    const int2 range = __ldg(ranges + blockIdx.x);
    const int n0 = range.x, n1 = range.y, tid = threadIdx.x;
    tile_setup(T, X, Y, Z, F, n0, n1, p, cap);
    const float fmax = __uint_as_float(T.fmax_bits);
    if (!(fmax > 0.f)) return;                                         // nothing to spread
    const bool tiled = T.enabled != 0 && fmax < 3.0e38f;
    const int e0 = T.e[0], e1 = T.e[1], ncell = tiled ? e0 * e1 * T.e[2] : 0;
    // |tile value| <= n_nodes * max W * max|F| = bound; scale = 2^k with bound * scale < 2^30
    const int k = max(-100, min(100, 29 - ilogbf(0.125f * (float)(n1 - n0) * fmax)));
    const float scale = tiled ? ldexpf(1.0f, k) : 1.0f, inv_scale = ldexpf(1.0f, -k);
    for (int t = tid; t < ncell; t += IB_THREADS) {
        tile[t] = 0; tile[cap + t] = 0; tile[2 * cap + t] = 0;
    }
    const int sub = tid & (LANES_PER_NODE - 1), ox = sub & 3, oy = sub >> 2;
    for (int c0 = n0; c0 < n1; c0 += IB_CHUNK) {
        __syncthreads();
        if (tid < IB_CHUNK && c0 + tid < n1) {
            const int m = c0 + tid;
            chunk_record(ch, T, tiled, tid, __ldg(X + m), __ldg(Y + m), __ldg(Z + m));
            const float4 Fm = __ldg(F + m);
            rF[tid] = Fm.x * scale; rF[IB_CHUNK + tid] = Fm.y * scale; rF[2 * IB_CHUNK + tid] = Fm.z * scale;
        }
        __syncthreads();
        const int cnt = min(IB_CHUNK, n1 - c0);
        for (int r = tid / LANES_PER_NODE; r < cnt; r += IB_GROUPS) {
            const Axis ax = chunk_axis(ch, 0, r), ay = chunk_axis(ch, 1, r), az = chunk_axis(ch, 2, r);
            const float Fx = rF[r], Fy = rF[IB_CHUNK + r], Fz = rF[2 * IB_CHUNK + r];
            const float wxy = weight_of(ax, ox) * weight_of(ay, oy);
            if (tiled) {
                const int tx = ax.base + ox, ty = ay.base + oy;
                if (tx < T.lo[0] || tx >= T.hi[0] || ty < T.lo[1] || ty >= T.hi[1]) continue;
#pragma unroll
                for (int oz = 0; oz < 4; ++oz) {
                    const int tz = az.base + oz;
                    if (tz < T.lo[2] || tz >= T.hi[2]) continue;
                    const float W = wxy * weight_of(az, oz);
                    const int t = (tz * e1 + ty) * e0 + tx;
                    atomicAdd(tile + t, __float2int_rn(W * Fx));
                    atomicAdd(tile + cap + t, __float2int_rn(W * Fy));
                    atomicAdd(tile + 2 * cap + t, __float2int_rn(W * Fz));
                }
            } else {
                const int qx = wrap_index(ax.base + ox, p.nx, p.wall[0]);
                const int qy = wrap_index(ay.base + oy, p.ny, p.wall[1]);
                if (qx < 0 || qy < 0) continue;
#pragma unroll
                for (int oz = 0; oz < 4; ++oz) {
                    const int qz = wrap_index(az.base + oz, p.nz, p.wall[2]);
                    if (qz < 0) continue;
                    const float W = wxy * weight_of(az, oz);
                    const int cell = qx + p.nx * (qy + p.ny * qz);
                    atomicAdd(g + cell, make_float4(W * Fx, W * Fy, W * Fz, 0.f));
                    mark_segment(cell, seg_mask);
                }
            }
        }
    }
    if (!tiled) return;
    __syncthreads();
    for (int t = tid; t < ncell; t += IB_THREADS) {
        const int qx = tile[t], qy = tile[cap + t], qz = tile[2 * cap + t];
        if ((qx | qy | qz) != 0) {
            const Cell c = tile_cell(T, t, p);
            const int cell = c.i + p.nx * (c.j + p.ny * c.k);
            atomicAdd(g + cell, make_float4((float)qx * inv_scale, (float)qy * inv_scale, (float)qz * inv_scale, 0.f));
            mark_segment(cell, seg_mask);
        }
    }
}

// zero the cells of the segments the previous spread touched, and drop their activity bits:
// one thread per segment (a 128-byte line of the forcing field), one warp per mask word
__global__ void __launch_bounds__(256) clear_spread_kernel(float4* __restrict__ g, unsigned* __restrict__ seg_mask,
                                                           const int n_segs, const int cells) {
    const int seg = blockIdx.x * 256 + threadIdx.x;
    const int word = seg >> 5;
    const unsigned m = (seg < n_segs) ? seg_mask[word] : 0u;
    if (__ballot_sync(0xffffffffu, m != 0u) == 0u) return;
    if ((m >> (seg & 31)) & 1u) {
        const int c0 = seg * SEG;
#pragma unroll
        for (int c = 0; c < SEG; ++c)
            if (c0 + c < cells) g[c0 + c] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    __syncwarp();
    if ((seg & 31) == 0 && m != 0u) seg_mask[word] = 0u;
}

// S4 + S5: U_m = sum v phi phi phi (Eq. 33) with v = (sum c_i f_i + g/2)/rho of the state after
// lbm_step (G11), by a 16-lane shuffle reduction over the 4x4x4 stencil, then
// X_m += U_m in fp64.
__global__ void __launch_bounds__(IB_THREADS) interpolate_mesh_kernel(
    double* __restrict__ X, double* __restrict__ Y, double* __restrict__ Z, float4* __restrict__ U,
    const int2* __restrict__ ranges, const float* __restrict__ src, const float4* __restrict__ g,
    int* __restrict__ counters, const LbmParams p, const int cap) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ MeshTile T;
    float* tile = reinterpret_cast<float*>(smem_raw);                  // [3][cap] velocity
    Chunk ch;
    ch.b = reinterpret_cast<int*>(tile + 3 * (size_t)cap);
    ch.sc = reinterpret_cast<float*>(ch.b + 3 * IB_CHUNK);
    unsigned short* list = reinterpret_cast<unsigned short*>(ch.sc + 6 * IB_CHUNK);   // [cap] needed tile cells
    const int2 range = __ldg(ranges + blockIdx.x);
    const int n0 = range.x, n1 = range.y, tid = threadIdx.x;
    tile_setup(T, X, Y, Z, nullptr, n0, n1, p, cap);
    const bool tiled = T.enabled != 0;
    const int e0 = T.e[0], e1 = T.e[1], ncell = tiled ? e0 * e1 * T.e[2] : 0;
    if (tiled) {
        unsigned* need = reinterpret_cast<unsigned*>(tile);           // marks live in the x plane of the tile
        for (int t = tid; t < ncell; t += IB_THREADS) need[t] = 0u;
        __syncthreads();
        for (int m = n0 + tid; m < n1; m += IB_THREADS) {             // the 4^3 cells each node needs
            const int bx = (int)floor(X[m]) - 1 - T.o[0], by = (int)floor(Y[m]) - 1 - T.o[1],
                      bz = (int)floor(Z[m]) - 1 - T.o[2];
            for (int oz = 0; oz < 4; ++oz) {
                const int tz = bz + oz;
                if (tz < T.lo[2] || tz >= T.hi[2]) continue;
                for (int oy = 0; oy < 4; ++oy) {
                    const int ty = by + oy;
                    if (ty < T.lo[1] || ty >= T.hi[1]) continue;
                    const int row = (tz * e1 + ty) * e0;
#pragma unroll
                    for (int ox = 0; ox < 4; ++ox) {
                        const int tx = bx + ox;
                        if (tx >= T.lo[0] && tx < T.hi[0]) need[row + tx] = 1u;
                    }
                }
            }
        }
        __syncthreads();
        // compact the needed cells so that every lane of the moment pass has a cell
        for (int t0 = 0; t0 < ncell; t0 += IB_THREADS) {
            const int t = t0 + tid;
            const bool want = t < ncell && need[t] != 0u;
            const unsigned vote = __ballot_sync(0xffffffffu, want);
            int base = 0;
            if ((tid & 31) == 0 && vote) base = atomicAdd(&T.n_need, __popc(vote));
            base = __shfl_sync(0xffffffffu, base, 0);
            if (want) list[base + __popc(vote & ((1u << (tid & 31)) - 1u))] = (unsigned short)t;
        }
        __syncthreads();
        const int n_need = T.n_need;
        for (int e = tid; e < n_need; e += IB_THREADS) {
            const int t = list[e];
            const float4 v = cell_macros(src, g, p, tile_cell(T, t, p));
            tile[t] = v.x; tile[cap + t] = v.y; tile[2 * cap + t] = v.z;
        }
    }
    const int sub = tid & (LANES_PER_NODE - 1), ox = sub & 3, oy = sub >> 2;
    for (int c0 = n0; c0 < n1; c0 += IB_CHUNK) {
        __syncthreads();
        if (tid < IB_CHUNK && c0 + tid < n1) {
            const int m = c0 + tid;
            chunk_record(ch, T, tiled, tid, X[m], Y[m], Z[m]);
        }
        __syncthreads();
        const int cnt = min(IB_CHUNK, n1 - c0);
        // the 16 lanes of a node iterate together: r is the same for a whole half-warp
        for (int r = tid / LANES_PER_NODE; r < cnt; r += IB_GROUPS) {
            const Axis ax = chunk_axis(ch, 0, r), ay = chunk_axis(ch, 1, r), az = chunk_axis(ch, 2, r);
            const float wxy = weight_of(ax, ox) * weight_of(ay, oy);
            float ux = 0.f, uy = 0.f, uz = 0.f;
            if (tiled) {
                const int tx = ax.base + ox, ty = ay.base + oy;
                if (tx >= T.lo[0] && tx < T.hi[0] && ty >= T.lo[1] && ty < T.hi[1]) {
#pragma unroll
                    for (int oz = 0; oz < 4; ++oz) {
                        const int tz = az.base + oz;
                        if (tz < T.lo[2] || tz >= T.hi[2]) continue;
                        const float W = wxy * weight_of(az, oz);
                        const int t = (tz * e1 + ty) * e0 + tx;
                        ux = fmaf(W, tile[t], ux);
                        uy = fmaf(W, tile[cap + t], uy);
                        uz = fmaf(W, tile[2 * cap + t], uz);
                    }
                }
            } else {
                const int qx = wrap_index(ax.base + ox, p.nx, p.wall[0]);
                const int qy = wrap_index(ay.base + oy, p.ny, p.wall[1]);
                if (qx >= 0 && qy >= 0) {
                    for (int oz = 0; oz < 4; ++oz) {
                        const int qz = wrap_index(az.base + oz, p.nz, p.wall[2]);
                        if (qz < 0) continue;
                        const float W = wxy * weight_of(az, oz);
                        Cell c;
                        c.i = qx; c.j = qy; c.k = qz;
                        const float4 v = cell_macros(src, g, p, c);
                        ux = fmaf(W, v.x, ux);
                        uy = fmaf(W, v.y, uy);
                        uz = fmaf(W, v.z, uz);
                    }
                }
            }
            const unsigned half = 0xffffu << (threadIdx.x & 16);
#pragma unroll
            for (int o = LANES_PER_NODE / 2; o > 0; o >>= 1) {
                ux += __shfl_xor_sync(half, ux, o);
                uy += __shfl_xor_sync(half, uy, o);
                uz += __shfl_xor_sync(half, uz, o);
            }
            if (sub == 0) {
                const int m = c0 + r;
                U[m] = make_float4(ux, uy, uz, 0.f);
                const double xn = X[m] + (double)ux, yn = Y[m] + (double)uy, zn = Z[m] + (double)uz;
                X[m] = xn; Y[m] = yn; Z[m] = zn;
                // halfway bounce-back walls lie at -1/2 and n - 1/2, on-site velocity walls at 0 and n - 1
                const double m0 = p.wall[0] == PLB_WALL_HH ? 0.0 : 0.5, m1 = p.wall[1] == PLB_WALL_HH ? 0.0 : 0.5,
                             m2 = p.wall[2] == PLB_WALL_HH ? 0.0 : 0.5;
                const bool left = (p.wall[0] && (xn < -m0 || xn > (double)(p.nx - 1) + m0)) ||
                                  (p.wall[1] && (yn < -m1 || yn > (double)(p.ny - 1) + m1)) ||
                                  (p.wall[2] && (zn < -m2 || zn > (double)(p.nz - 1) + m2));
                if (left) atomicOr(counters + 1, STATUS_NODE_LEFT);
            }
        }
    }
}

// positions: device SoA <-> AoS staging buffer (so host transfers are one contiguous copy)
__global__ void __launch_bounds__(256) nodes_transpose_kernel(double* __restrict__ X, double* __restrict__ Y,
                                                              double* __restrict__ Z, double* __restrict__ aos,
                                                              const long n, const bool to_aos) {
    const long t = blockIdx.x * 256L + threadIdx.x;
    if (t >= 3 * n) return;
    const long m = t / 3;
    const int d = (int)(t - 3 * m);
    double* comp = d == 0 ? X : (d == 1 ? Y : Z);
    if (to_aos) aos[t] = comp[m];
    else        comp[m] = aos[t];
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
    force_init_kernel<<<(unsigned)((c->n_nodes + 255) / 256), 256, 0, c->stream>>>(c->F, c->n_nodes, sigma, seed,
                                                                                  (unsigned)step);
    c->launches++;
    if (c->n_edges) {
        edge_force_kernel<<<(unsigned)((c->n_edges + 255) / 256), 256, 0, c->stream>>>(
            c->X[0], c->X[1], c->X[2], c->edges, c->edge_prm, c->F, c->n_edges, c->counters);
        c->launches++;
    }
    if (c->n_cons) {
        constraint_force_kernel<<<(unsigned)c->n_cons, CON_THREADS, 0, c->stream>>>(
            c->X[0], c->X[1], c->X[2], c->tris, c->tri_S0, c->cons, c->F);
        c->launches++;
    }
    return cuda_check(cudaGetLastError(), "membrane force kernels");
}

int launch_clear_spread(Ctx* c, float4* g) {
    clear_spread_kernel<<<(unsigned)((c->n_segs + 255) / 256), 256, 0, c->stream>>>(g, c->seg_mask, (int)c->n_segs,
                                                                                  c->prm.cells);
    c->launches++;
    return cuda_check(cudaGetLastError(), "clear_spread_kernel");
}

static size_t spread_smem(int cap) { return (size_t)cap * 12 + (size_t)IB_CHUNK * 48; }
static size_t interp_smem(int cap) { return (size_t)cap * 12 + (size_t)IB_CHUNK * 36 + (((size_t)cap * 2 + 15) & ~(size_t)15); }

// Largest tile (in cells) both kernels can hold with at least one block per SM; a tile cell index
// must also fit the 16-bit entries of the interpolation's compact list.
int ib_max_tile_cap() {
    const size_t budget = 200 * 1024;
    const size_t cap = (budget - (size_t)IB_CHUNK * 48 - 64) / 14;
    return (int)(cap < 65535 ? cap : 65535);
}

int launch_spread(Ctx* c, float4* g) {
    if (c->n_nodes == 0) return PLB_OK;
    const size_t smem = spread_smem(c->tile_cap);
    int rc = cuda_check(cudaFuncSetAttribute(spread_mesh_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem),
                        "cudaFuncSetAttribute(spread_mesh_kernel)");
    if (rc) return rc;
    spread_mesh_kernel<<<(unsigned)c->n_ranges, IB_THREADS, smem, c->stream>>>(
        c->X[0], c->X[1], c->X[2], c->F, c->ranges, g, c->seg_mask, c->prm, c->tile_cap);
    c->launches++;
    return cuda_check(cudaGetLastError(), "spread_mesh_kernel");
}

int launch_interpolate_advance(Ctx* c) {
    if (c->n_nodes == 0) return PLB_OK;
    const size_t smem = interp_smem(c->tile_cap);
    int rc = cuda_check(cudaFuncSetAttribute(interpolate_mesh_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem),
                        "cudaFuncSetAttribute(interpolate_mesh_kernel)");
    if (rc) return rc;
    const float4* g = (c->g_last_mode == FORCE_NONE) ? nullptr : c->g_last;
    interpolate_mesh_kernel<<<(unsigned)c->n_ranges, IB_THREADS, smem, c->stream>>>(
        c->X[0], c->X[1], c->X[2], c->U, c->ranges, c->f[c->cur], g, c->counters, c->prm, c->tile_cap);
    c->launches++;
    return cuda_check(cudaGetLastError(), "interpolate_mesh_kernel");
}

int launch_nodes_transpose(Ctx* c, bool to_aos) {
    if (c->n_nodes == 0) return PLB_OK;
    nodes_transpose_kernel<<<(unsigned)((3 * c->n_nodes + 255) / 256), 256, 0, c->stream>>>(
        c->X[0], c->X[1], c->X[2], c->stage, c->n_nodes, to_aos);
    c->launches++;
    return cuda_check(cudaGetLastError(), "nodes_transpose_kernel");
}

int launch_philox(cudaStream_t s, long n, const unsigned* ctr, const unsigned* key, unsigned* out) {
    if (n <= 0) return PLB_OK;
    philox_kernel<<<(unsigned)((n + 127) / 128), 128, 0, s>>>(n, (const uint4*)ctr, (const uint2*)key, (uint4*)out);
    return cuda_check(cudaGetLastError(), "philox_kernel");
}

}  // namespace plb
