// ib.cu -- immersed-boundary and membrane kernels (Eq. 2-3, section 3.4.2 Eq. 31-36).
//
// Node data: positions SoA fp64 (unwrapped), forces / node velocities float4 AoS.
// The forcing field is float4 per cell so that the spread is one 128-bit vector atomic per
// (node, cell) pair (red.global.add.v4.f32, sm_90+).
#include "plb_internal.cuh"

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

// S2 + S4 share the mapping: 16 lanes per node, lane = (ox, oy), loop over oz.  Four lanes with
// the same (oy, oz) touch four consecutive cells = 64 contiguous bytes of the float4 field.
constexpr int LANES_PER_NODE = 16;

// set the activity bit of a segment; whoever sets it first appends the segment to the list
__device__ __forceinline__ void mark_segment(const int seg, unsigned* __restrict__ seg_mask, int* __restrict__ seg_list,
                                             int* __restrict__ counters) {
    const unsigned bit = 1u << (seg & 31);
    unsigned* word = seg_mask + (seg >> 5);
    if ((*(volatile unsigned*)word & bit) == 0u && (atomicOr(word, bit) & bit) == 0u)
        seg_list[atomicAdd(counters, 1)] = seg;
}

// S2: g_ijk += F_m phi phi phi (Eq. 34).  Also records which 32-cell segments were touched.
__global__ void __launch_bounds__(256) spread_kernel(const double* __restrict__ X, const double* __restrict__ Y,
                                                     const double* __restrict__ Z, const float4* __restrict__ F,
                                                     const long n_nodes, float4* __restrict__ g,
                                                     unsigned* __restrict__ seg_mask, int* __restrict__ seg_list,
                                                     int* __restrict__ counters, const LbmParams p) {
    const long t = blockIdx.x * 256L + threadIdx.x;
    const long m = t / LANES_PER_NODE;
    if (m >= n_nodes) return;
    const int sub = (int)(t % LANES_PER_NODE), ox = sub & 3, oy = sub >> 2;
    const Axis ax = axis_of(__ldg(X + m)), ay = axis_of(__ldg(Y + m)), az = axis_of(__ldg(Z + m));
    const float4 Fm = __ldg(F + m);
    const int qx = wrap_index(ax.base + ox, p.nx, p.wall[0]);
    const int qy = wrap_index(ay.base + oy, p.ny, p.wall[1]);
    if (qx < 0 || qy < 0) return;
    const float wxy = weight_of(ax, ox) * weight_of(ay, oy);
#pragma unroll
    for (int oz = 0; oz < 4; ++oz) {
        const int qz = wrap_index(az.base + oz, p.nz, p.wall[2]);
        if (qz < 0) continue;
        const float W = wxy * weight_of(az, oz);
        const int cell = qx + p.nx * (qy + p.ny * qz);
        atomicAdd(g + cell, make_float4(W * Fm.x, W * Fm.y, W * Fm.z, 0.f));
        mark_segment(cell >> SEG_SHIFT, seg_mask, seg_list, counters);
    }
}

// zero the cells of the segments the previous spread touched, and drop their activity bits
__global__ void __launch_bounds__(256) clear_spread_kernel(float4* __restrict__ g, unsigned* __restrict__ seg_mask,
                                                           const int* __restrict__ seg_list,
                                                           const int* __restrict__ counters, const int cells) {
    const int sub = threadIdx.x & (SEG - 1);
    const int group = (blockIdx.x * 256 + threadIdx.x) >> SEG_SHIFT;
    const int n_groups = (gridDim.x * 256) >> SEG_SHIFT;
    const int n_active = __ldg(counters);
    for (int s = group; s < n_active; s += n_groups) {
        const int seg = seg_list[s];
        const int idx = seg * SEG + sub;
        if (idx < cells) g[idx] = make_float4(0.f, 0.f, 0.f, 0.f);
        if (sub == 0) seg_mask[seg >> 5] = 0u;        // every set bit of the word is in the list
    }
}

// S4 + S5: U_m = sum v phi phi phi (Eq. 33) by a 16-lane shuffle reduction over the 4x4x4
// stencil, then X_m += U_m in fp64.
__global__ void __launch_bounds__(256) interpolate_advance_kernel(double* __restrict__ X, double* __restrict__ Y,
                                                                  double* __restrict__ Z, float4* __restrict__ U,
                                                                  const long n_nodes, const float4* __restrict__ vel,
                                                                  int* __restrict__ counters, const LbmParams p) {
    const long t = blockIdx.x * 256L + threadIdx.x;
    const long m = t / LANES_PER_NODE;
    const bool live = m < n_nodes;                      // dead lanes still take part in the shuffles
    const int sub = (int)(t % LANES_PER_NODE), ox = sub & 3, oy = sub >> 2;
    const double xm = live ? X[m] : 0.0, ym = live ? Y[m] : 0.0, zm = live ? Z[m] : 0.0;
    const Axis ax = axis_of(xm), ay = axis_of(ym), az = axis_of(zm);
    const int qx = wrap_index(ax.base + ox, p.nx, p.wall[0]);
    const int qy = wrap_index(ay.base + oy, p.ny, p.wall[1]);
    float ux = 0.f, uy = 0.f, uz = 0.f;
    if (live && qx >= 0 && qy >= 0) {
        const float wxy = weight_of(ax, ox) * weight_of(ay, oy);
#pragma unroll
        for (int oz = 0; oz < 4; ++oz) {
            const int qz = wrap_index(az.base + oz, p.nz, p.wall[2]);
            if (qz < 0) continue;
            const float W = wxy * weight_of(az, oz);
            const float4 v = vel[qx + p.nx * (qy + p.ny * qz)];
            ux = fmaf(W, v.x, ux);
            uy = fmaf(W, v.y, uy);
            uz = fmaf(W, v.z, uz);
        }
    }
#pragma unroll
    for (int o = LANES_PER_NODE / 2; o > 0; o >>= 1) {
        ux += __shfl_xor_sync(0xffffffffu, ux, o);
        uy += __shfl_xor_sync(0xffffffffu, uy, o);
        uz += __shfl_xor_sync(0xffffffffu, uz, o);
    }
    if (live && sub == 0) {
        U[m] = make_float4(ux, uy, uz, 0.f);
        const double xn = xm + (double)ux, yn = ym + (double)uy, zn = zm + (double)uz;
        X[m] = xn; Y[m] = yn; Z[m] = zn;
        const bool left = (p.wall[0] && (xn < -0.5 || xn > (double)p.nx - 0.5)) ||
                          (p.wall[1] && (yn < -0.5 || yn > (double)p.ny - 0.5)) ||
                          (p.wall[2] && (zn < -0.5 || zn > (double)p.nz - 0.5));
        if (left) atomicOr(counters + 1, STATUS_NODE_LEFT);
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
    return cuda_check(cudaGetLastError(), "edge_force_kernel");
}

int launch_clear_spread(Ctx* c, float4* g) {
    clear_spread_kernel<<<c->sm_count * 8, 256, 0, c->stream>>>(g, c->seg_mask, c->seg_list, c->counters, c->prm.cells);
    c->launches++;
    int rc = cuda_check(cudaGetLastError(), "clear_spread_kernel");
    if (rc) return rc;
    return cuda_check(cudaMemsetAsync(c->counters, 0, sizeof(int), c->stream), "reset segment counter");
}

int launch_spread(Ctx* c, float4* g) {
    if (c->n_nodes == 0) return PLB_OK;
    const long threads = c->n_nodes * LANES_PER_NODE;
    spread_kernel<<<(unsigned)((threads + 255) / 256), 256, 0, c->stream>>>(
        c->X[0], c->X[1], c->X[2], c->F, c->n_nodes, g, c->seg_mask, c->seg_list, c->counters, c->prm);
    c->launches++;
    return cuda_check(cudaGetLastError(), "spread_kernel");
}

int launch_interpolate_advance(Ctx* c) {
    if (c->n_nodes == 0) return PLB_OK;
    const long threads = c->n_nodes * LANES_PER_NODE;
    interpolate_advance_kernel<<<(unsigned)((threads + 255) / 256), 256, 0, c->stream>>>(
        c->X[0], c->X[1], c->X[2], c->U, c->n_nodes, c->vel, c->counters, c->prm);
    c->launches++;
    return cuda_check(cudaGetLastError(), "interpolate_advance_kernel");
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
