// lbm.cu -- D3Q19 BGK lattice-Boltzmann kernels (section 3.3, Eq. 15-21) for sm_100a.
//
// Storage: two fp32 lattices, SoA (population d of cell q at [d*cells + q]), holding
//     T_d(x) - w_d,
// where T is the POST-COLLISION ("pre-stream") state: streaming T gives the paper's f.
//     f_d(x) = T_d(x - c_d)                              (periodic wrap, L217)
//     f_d(x) = T_dbar(x) + 6 w_d (c_d . u_wall)           (x - c_d beyond a wall face: halfway
//                                                          bounce-back + Ladd term, rho_w = 1)
// so one fused kernel does pull-stream -> moments -> BGK + Guo forcing -> aligned store.
// The w_d shift keeps |stored value| ~ 1e-2 so that fp32 holds |d rho| <= 1e-6.
#include "plb_internal.cuh"

namespace plb {

struct Cell {
    int i, j, k;
};

__device__ __forceinline__ Cell cell_of(int idx, const LbmParams& p) {
    Cell c;
    const unsigned t = (unsigned)idx / (unsigned)p.nx;
    c.i = (int)((unsigned)idx - t * (unsigned)p.nx);
    c.k = (int)(t / (unsigned)p.ny);
    c.j = (int)(t - (unsigned)c.k * (unsigned)p.ny);
    return c;
}

// Pull the 19 streamed populations (minus w_d) of cell (i,j,k) out of the pre-stream lattice.
__device__ __forceinline__ void pull19(const float* __restrict__ src, const LbmParams& p, const Cell c,
                                       const int idx, float h[Q]) {
    const int nx = p.nx, ny = p.ny, nz = p.nz;
    const size_t N = (size_t)p.cells;
    const bool xlo = c.i == 0, xhi = c.i == nx - 1;
    const bool ylo = c.j == 0, yhi = c.j == ny - 1;
    const bool zlo = c.k == 0, zhi = c.k == nz - 1;
    // neighbour offsets with periodic wrap (a wall axis bounces instead, decided below)
    const int dxm = xlo ? nx - 1 : -1, dxp = xhi ? 1 - nx : 1;
    const int dym = (ylo ? ny - 1 : -1) * nx, dyp = (yhi ? 1 - ny : 1) * nx;
    const int dzm = (zlo ? nz - 1 : -1) * nx * ny, dzp = (zhi ? 1 - nz : 1) * nx * ny;
    const bool bxlo = p.wall[0] && xlo, bxhi = p.wall[0] && xhi;
    const bool bylo = p.wall[1] && ylo, byhi = p.wall[1] && yhi;
    const bool bzlo = p.wall[2] && zlo, bzhi = p.wall[2] && zhi;
#pragma unroll
    for (int d = 0; d < Q; ++d) {
        const int cx = CX(d), cy = CY(d), cz = CZ(d);
        // source cell x - c_d
        int off = 0;
        if (cx == 1) off += dxm;
        if (cx == -1) off += dxp;
        if (cy == 1) off += dym;
        if (cy == -1) off += dyp;
        if (cz == 1) off += dzm;
        if (cz == -1) off += dzp;
        // bounce-back: x - c_d lies beyond a wall face; z, y, x in this order so that x wins
        bool b = false;
        float corr = 0.f;
        if (cz == 1 && bzlo) { b = true; corr = p.corr[2][0][d]; }
        if (cz == -1 && bzhi) { b = true; corr = p.corr[2][1][d]; }
        if (cy == 1 && bylo) { b = true; corr = p.corr[1][0][d]; }
        if (cy == -1 && byhi) { b = true; corr = p.corr[1][1][d]; }
        if (cx == 1 && bxlo) { b = true; corr = p.corr[0][0][d]; }
        if (cx == -1 && bxhi) { b = true; corr = p.corr[0][1][d]; }
        if (b) h[d] = __ldg(src + (size_t)OPP(d) * N + idx) + corr;
        else   h[d] = __ldg(src + (size_t)d * N + (idx + off));
    }
}

// delta rho = sum h_d, j = sum c_d h_d (Eq. 17-18; sum_d w_d c_d = 0 so the shift drops out of j)
__device__ __forceinline__ void moments(const float h[Q], float& drho, float& jx, float& jy, float& jz) {
    // pairwise sums keep the fp32 rounding small and symmetric
    const float a01p = h[0] + h[1], a23p = h[2] + h[3], a45p = h[4] + h[5];
    const float s6 = (h[6] + h[11]) + (h[7] + h[10]);      // xy diagonals
    const float s8 = (h[8] + h[13]) + (h[9] + h[12]);      // xz diagonals
    const float s14 = (h[14] + h[17]) + (h[15] + h[16]);   // yz diagonals
    drho = ((a01p + a23p) + (a45p + h[18])) + ((s6 + s8) + s14);
    jx = (h[0] - h[1]) + (((h[6] - h[11]) + (h[7] - h[10])) + ((h[8] - h[13]) + (h[9] - h[12])));
    jy = (h[2] - h[3]) + (((h[6] - h[11]) - (h[7] - h[10])) + ((h[14] - h[17]) + (h[15] - h[16])));
    jz = (h[4] - h[5]) + (((h[8] - h[13]) - (h[9] - h[12])) + ((h[14] - h[17]) - (h[15] - h[16])));
}

// BGK relaxation (Eq. 16) towards f_eq(rho, v) (Eq. 20) with v = u + g/(2 rho) (L201) plus the
// Guo term (Eq. 19 in the form S_d = (1 - 1/2tau) w_d [3 (c_d - v).g + 9 (c_d.v)(c_d.g)],
// DESIGN.md G3), all on the shifted populations:  h_eq,d = w_d [drho + rho (3 c.v + 4.5 (c.v)^2 - 1.5 v^2)].
template <bool FORCED>
__device__ __forceinline__ void collide(float h[Q], const float gx, const float gy, const float gz,
                                        const float omega, const float pref) {
    float drho, jx, jy, jz;
    moments(h, drho, jx, jy, jz);
    const float rho = 1.0f + drho;
    const float inv = 1.0f / rho;
    float vx, vy, vz;
    if (FORCED) {
        vx = (jx + 0.5f * gx) * inv; vy = (jy + 0.5f * gy) * inv; vz = (jz + 0.5f * gz) * inv;
    } else {
        vx = jx * inv; vy = jy * inv; vz = jz * inv;
    }
    const float vv15 = 1.5f * (vx * vx + vy * vy + vz * vz);
    const float vg3 = 3.0f * (vx * gx + vy * gy + vz * gz);
#pragma unroll
    for (int d = 0; d < Q; ++d) {
        const float cx = (float)CX(d), cy = (float)CY(d), cz = (float)CZ(d);
        const float cv = cx * vx + cy * vy + cz * vz;
        const float heq = WGT(d) * (drho + rho * (3.0f * cv + 4.5f * cv * cv - vv15));
        float out = h[d] + omega * (heq - h[d]);
        if (FORCED) {
            const float cg = cx * gx + cy * gy + cz * gz;
            out += pref * WGT(d) * (3.0f * cg - vg3 + 9.0f * cv * cg);
        }
        h[d] = out;
    }
}

// ---------------------------------------------------------------------------------------------
// S3: fused pull-stream + collide + boundary kernel.  One thread per cell, one warp per
// 32-cell segment; loads along x are unit-stride, stores are aligned and coalesced.
// ---------------------------------------------------------------------------------------------
template <int MODE>
__global__ void __launch_bounds__(256) lbm_step_kernel(const float* __restrict__ src, float* __restrict__ dst,
                                                       const float4* __restrict__ g,
                                                       const int* __restrict__ seg_flag, const LbmParams p) {
    const int idx = blockIdx.x * 256 + threadIdx.x;
    if (idx >= p.cells) return;
    const Cell c = cell_of(idx, p);
    float h[Q];
    pull19(src, p, c, idx, h);
    bool forced = false;
    float4 g4 = make_float4(0.f, 0.f, 0.f, 0.f);
    if (MODE == FORCE_DENSE) {
        g4 = __ldg(g + idx);
        forced = true;
    } else if (MODE == FORCE_SPARSE) {
        if (__ldg(seg_flag + (idx >> SEG_SHIFT))) {      // warp-uniform
            g4 = __ldg(g + idx);
            forced = true;
        }
    }
    if (forced) collide<true>(h, g4.x, g4.y, g4.z, p.omega, p.pref);
    else        collide<false>(h, 0.f, 0.f, 0.f, p.omega, p.pref);
    const size_t N = (size_t)p.cells;
#pragma unroll
    for (int d = 0; d < Q; ++d) dst[(size_t)d * N + idx] = h[d];
}

// rho and v = (j + g_last/2)/rho of the streamed state (what the next step will collide)
template <int MODE>
__global__ void __launch_bounds__(256) macros_kernel(const float* __restrict__ src, const float4* __restrict__ g,
                                                     const int* __restrict__ seg_flag, float* __restrict__ rho_out,
                                                     float* __restrict__ u_out, const LbmParams p) {
    const int idx = blockIdx.x * 256 + threadIdx.x;
    if (idx >= p.cells) return;
    const Cell c = cell_of(idx, p);
    float h[Q];
    pull19(src, p, c, idx, h);
    float drho, jx, jy, jz;
    moments(h, drho, jx, jy, jz);
    float4 g4 = make_float4(0.f, 0.f, 0.f, 0.f);
    if (MODE == FORCE_DENSE) g4 = __ldg(g + idx);
    if (MODE == FORCE_SPARSE && __ldg(seg_flag + (idx >> SEG_SHIFT))) g4 = __ldg(g + idx);
    const float rho = 1.0f + drho, inv = 1.0f / rho;
    if (rho_out) rho_out[idx] = rho;
    if (u_out) {
        const size_t N = (size_t)p.cells;
        u_out[idx] = (jx + 0.5f * g4.x) * inv;
        u_out[N + idx] = (jy + 0.5f * g4.y) * inv;
        u_out[2 * N + idx] = (jz + 0.5f * g4.z) * inv;
    }
}

// The same moments, only over the segments the last ib_spread touched (the 4^3 supports of the
// nodes), written as float4 (vx, vy, vz, rho) for the interpolation gather.
template <int MODE>
__global__ void __launch_bounds__(256) sparse_moments_kernel(const float* __restrict__ src,
                                                             const float4* __restrict__ g,
                                                             const int* __restrict__ seg_list,
                                                             const int* __restrict__ counters,
                                                             float4* __restrict__ vel, const LbmParams p) {
    const int lane = threadIdx.x & 31;
    const int warp = (blockIdx.x * 256 + threadIdx.x) >> 5;
    const int n_warps = (gridDim.x * 256) >> 5;
    const int n_active = __ldg(counters);
    for (int s = warp; s < n_active; s += n_warps) {
        const int idx = __ldg(seg_list + s) * SEG + lane;
        if (idx >= p.cells) continue;
        const Cell c = cell_of(idx, p);
        float h[Q];
        pull19(src, p, c, idx, h);
        float drho, jx, jy, jz;
        moments(h, drho, jx, jy, jz);
        float4 g4 = make_float4(0.f, 0.f, 0.f, 0.f);
        if (MODE != FORCE_NONE) g4 = __ldg(g + idx);
        const float rho = 1.0f + drho, inv = 1.0f / rho;
        vel[idx] = make_float4((jx + 0.5f * g4.x) * inv, (jy + 0.5f * g4.y) * inv, (jz + 0.5f * g4.z) * inv, rho);
    }
}

// ---------------------------------------------------------------------------------------------
// initialisation / checkpoint kernels (off the timed path).  They write the pre-stream state T:
//   T_d(x) = f_d(x + c_d)                               (interior / periodic)
//   T_d(x) = f_dbar(x) - 6 w_dbar (c_dbar . u_wall)      (link d leaves through a wall face)
// ---------------------------------------------------------------------------------------------
struct Target {
    int idx;      // cell whose f is wanted
    int d;        // which population of that cell
    float corr;   // to subtract
};

template <int D>
__device__ __forceinline__ Target pre_stream_target(const LbmParams& p, const Cell c, const int idx) {
    constexpr int cx = CX(D), cy = CY(D), cz = CZ(D);
    const int nx = p.nx, ny = p.ny, nz = p.nz;
    int ti = c.i + cx, tj = c.j + cy, tk = c.k + cz;
    bool b = false;
    float corr = 0.f;
    // link D from x leaves through ...; z, y, x order so that x wins (corner rule)
    if (tk < 0) { if (p.wall[2]) { b = true; corr = p.corr[2][0][OPP(D)]; } else tk += nz; }
    if (tk >= nz) { if (p.wall[2]) { b = true; corr = p.corr[2][1][OPP(D)]; } else tk -= nz; }
    if (tj < 0) { if (p.wall[1]) { b = true; corr = p.corr[1][0][OPP(D)]; } else tj += ny; }
    if (tj >= ny) { if (p.wall[1]) { b = true; corr = p.corr[1][1][OPP(D)]; } else tj -= ny; }
    if (ti < 0) { if (p.wall[0]) { b = true; corr = p.corr[0][0][OPP(D)]; } else ti += nx; }
    if (ti >= nx) { if (p.wall[0]) { b = true; corr = p.corr[0][1][OPP(D)]; } else ti -= nx; }
    Target t;
    if (b) { t.idx = idx; t.d = OPP(D); t.corr = corr; }
    else   { t.idx = ti + nx * (tj + ny * tk); t.d = D; t.corr = 0.f; }
    return t;
}

// h_eq,d = f_eq,d - w_d of Eq. 20 at (rho, u), plus the seeded population noise
__device__ __forceinline__ float init_value(const int d, const int cell, const float* __restrict__ rho_in,
                                            const float* __restrict__ u_in, const size_t N, const float amp,
                                            const unsigned long long seed) {
    const float rho = rho_in ? __ldg(rho_in + cell) : 1.0f;
    const float ux = u_in ? __ldg(u_in + cell) : 0.f;
    const float uy = u_in ? __ldg(u_in + N + cell) : 0.f;
    const float uz = u_in ? __ldg(u_in + 2 * N + cell) : 0.f;
    const float cu = (float)CX(d) * ux + (float)CY(d) * uy + (float)CZ(d) * uz;
    const float wd = d < 6 ? (1.0f / 18.0f) : (d < 18 ? (1.0f / 36.0f) : (1.0f / 3.0f));
    float v = wd * ((rho - 1.0f) + rho * (3.0f * cu + 4.5f * cu * cu - 1.5f * (ux * ux + uy * uy + uz * uz)));
    if (amp > 0.f) {
        const uint4 r = noise_words(seed, (unsigned long long)cell * Q + (unsigned long long)d, 0u, 1u);
        v += amp * (2.0f * uniform01(r.x) - 1.0f);
    }
    return v;
}

template <int D>
__device__ __forceinline__ void init_one(float* __restrict__ dst, const LbmParams& p, const Cell c, const int idx,
                                         const float* rho_in, const float* u_in, const float amp,
                                         const unsigned long long seed) {
    const Target t = pre_stream_target<D>(p, c, idx);
    dst[(size_t)D * p.cells + idx] = init_value(t.d, t.idx, rho_in, u_in, (size_t)p.cells, amp, seed) - t.corr;
    if constexpr (D + 1 < Q) init_one<D + 1>(dst, p, c, idx, rho_in, u_in, amp, seed);
}

__global__ void __launch_bounds__(256) set_equilibrium_kernel(float* __restrict__ dst, const float* __restrict__ rho_in,
                                                              const float* __restrict__ u_in, const float amp,
                                                              const unsigned long long seed, const LbmParams p) {
    const int idx = blockIdx.x * 256 + threadIdx.x;
    if (idx >= p.cells) return;
    init_one<0>(dst, p, cell_of(idx, p), idx, rho_in, u_in, amp, seed);
}

template <int D>
__device__ __forceinline__ void write_one(float* __restrict__ dst, const float* __restrict__ f, const LbmParams& p,
                                          const Cell c, const int idx) {
    const Target t = pre_stream_target<D>(p, c, idx);
    const float wd = WGT(D);
    dst[(size_t)D * p.cells + idx] = (__ldg(f + (size_t)t.d * p.cells + t.idx) - wd) - t.corr;
    if constexpr (D + 1 < Q) write_one<D + 1>(dst, f, p, c, idx);
}

__global__ void __launch_bounds__(256) write_populations_kernel(float* __restrict__ dst, const float* __restrict__ f,
                                                                const LbmParams p) {
    const int idx = blockIdx.x * 256 + threadIdx.x;
    if (idx >= p.cells) return;
    write_one<0>(dst, f, p, cell_of(idx, p), idx);
}

__global__ void __launch_bounds__(256) read_populations_kernel(const float* __restrict__ src, float* __restrict__ f,
                                                               const LbmParams p) {
    const int idx = blockIdx.x * 256 + threadIdx.x;
    if (idx >= p.cells) return;
    float h[Q];
    pull19(src, p, cell_of(idx, p), idx, h);
#pragma unroll
    for (int d = 0; d < Q; ++d) f[(size_t)d * p.cells + idx] = h[d] + WGT(d);
}

// ---------------------------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------------------------
static inline int grid_cells(const Ctx* c) { return (c->prm.cells + 255) / 256; }

int launch_set_equilibrium(Ctx* c, const float* d_rho, const float* d_u, float amp, unsigned long long seed) {
    set_equilibrium_kernel<<<grid_cells(c), 256, 0, c->stream>>>(c->f[c->cur], d_rho, d_u, amp, seed, c->prm);
    c->launches++;
    return cuda_check(cudaGetLastError(), "set_equilibrium_kernel");
}

int launch_lbm_step(Ctx* c, const float4* g, int mode) {
    const float* src = c->f[c->cur];
    float* dst = c->f[c->cur ^ 1];
    const int grid = grid_cells(c);
    if (mode == FORCE_NONE) lbm_step_kernel<FORCE_NONE><<<grid, 256, 0, c->stream>>>(src, dst, nullptr, nullptr, c->prm);
    else if (mode == FORCE_DENSE) lbm_step_kernel<FORCE_DENSE><<<grid, 256, 0, c->stream>>>(src, dst, g, nullptr, c->prm);
    else lbm_step_kernel<FORCE_SPARSE><<<grid, 256, 0, c->stream>>>(src, dst, g, c->seg_flag, c->prm);
    c->launches++;
    c->cur ^= 1;
    return cuda_check(cudaGetLastError(), "lbm_step_kernel");
}

int launch_read_macros(Ctx* c, float* d_rho, float* d_u) {
    const float* src = c->f[c->cur];
    const int grid = grid_cells(c);
    if (c->g_last_mode == FORCE_NONE || !c->g_last)
        macros_kernel<FORCE_NONE><<<grid, 256, 0, c->stream>>>(src, nullptr, nullptr, d_rho, d_u, c->prm);
    else if (c->g_last_mode == FORCE_DENSE)
        macros_kernel<FORCE_DENSE><<<grid, 256, 0, c->stream>>>(src, c->g_last, nullptr, d_rho, d_u, c->prm);
    else
        macros_kernel<FORCE_SPARSE><<<grid, 256, 0, c->stream>>>(src, c->g_last, c->seg_flag, d_rho, d_u, c->prm);
    c->launches++;
    return cuda_check(cudaGetLastError(), "macros_kernel");
}

int launch_sparse_moments(Ctx* c) {
    const float* src = c->f[c->cur];
    const int grid = c->sm_count * 8;
    if (c->g_last_mode == FORCE_NONE || !c->g_last)
        sparse_moments_kernel<FORCE_NONE><<<grid, 256, 0, c->stream>>>(src, nullptr, c->seg_list, c->counters, c->vel, c->prm);
    else
        sparse_moments_kernel<FORCE_DENSE><<<grid, 256, 0, c->stream>>>(src, c->g_last, c->seg_list, c->counters, c->vel, c->prm);
    c->launches++;
    return cuda_check(cudaGetLastError(), "sparse_moments_kernel");
}

int launch_read_populations(Ctx* c, float* d_f) {
    read_populations_kernel<<<grid_cells(c), 256, 0, c->stream>>>(c->f[c->cur], d_f, c->prm);
    c->launches++;
    return cuda_check(cudaGetLastError(), "read_populations_kernel");
}

int launch_write_populations(Ctx* c, const float* d_f) {
    write_populations_kernel<<<grid_cells(c), 256, 0, c->stream>>>(c->f[c->cur], d_f, c->prm);
    c->launches++;
    return cuda_check(cudaGetLastError(), "write_populations_kernel");
}

}  // namespace plb
