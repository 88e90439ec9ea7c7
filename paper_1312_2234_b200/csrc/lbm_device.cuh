// lbm_device.cuh -- device functions shared by the lattice kernels (lbm.cu) and the immersed-
// boundary kernels (ib.cu): cell indexing, the pull of the 19 streamed populations out of the
// pre-stream lattice, and their moments.
#pragma once
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

__host__ __device__ constexpr int CA(int a, int d) { return a == 0 ? CX(d) : (a == 1 ? CY(d) : CZ(d)); }

// Hecht-Harting on-site velocity wall (Eq. 23-30) on a cell of
// the face of axis A with inward normal n = sgn e_A and wall velocity vw: the populations with
// c.n = +1 did not arrive by streaming and are closed from the others,
//     rho = [sum_{c.n=0} f + 2 sum_{c.n=-1} f]/(1 - v.n),       f_n = f_-n + rho v.n/3,
//     f_{n + s t} = f_opp + rho (v.n + s v_t)/6 - s N_t,   N_t = (1/2) sum_{c.n=0} c_t f - rho v_t/3.
// Written on the shifted values h = f - w:  sum_{c.n=0} w + 2 sum_{c.n=-1} w = 2/3 + 2/6 = 1 and
// w_i = w_opp(i), so only the density needs the shift put back.
template <int A, int V, int COL>
__device__ __forceinline__ void hecht_harting_close(float (&h)[Q][V], const int sgn, const float* __restrict__ vw) {
    const float vn = (float)sgn * vw[A];
    float s0 = 0.f, sm = 0.f, T[3] = {0.f, 0.f, 0.f};
#pragma unroll
    for (int d = 0; d < Q; ++d) {
        const int ca = CA(A, d);
        if (ca == 0) {
            s0 += h[d][COL];
#pragma unroll
            for (int b = 0; b < 3; ++b)
                if (b != A && CA(b, d) != 0) T[b] += (float)CA(b, d) * h[d][COL];
        } else {
            sm += (ca == -sgn) ? h[d][COL] : 0.f;
        }
    }
    const float rho = (1.0f + (s0 + 2.0f * sm)) / (1.0f - vn);
    float N[3];
#pragma unroll
    for (int b = 0; b < 3; ++b) N[b] = 0.5f * T[b] - rho * vw[b] * (1.0f / 3.0f);
#pragma unroll
    for (int d = 0; d < Q; ++d) {
        const int ca = CA(A, d);
        if (ca == 0) continue;
        float val;
        int bt = -1;
#pragma unroll
        for (int b = 0; b < 3; ++b)
            if (b != A && CA(b, d) != 0) bt = b;
        if (bt < 0) val = h[OPP(d)][COL] + rho * vn * (1.0f / 3.0f);
        else {
            const float ct = (float)CA(bt, d);
            val = h[OPP(d)][COL] + rho * (vn + ct * vw[bt]) * (1.0f / 6.0f) - ct * N[bt];
        }
        if (ca == sgn) h[d][COL] = val;
    }
}

// Pull the 19 streamed populations (minus w_d) of cell (i,j,k) out of the pre-stream lattice
// into column COL of h.  Generic in the boundary kinds of all three axes.
template <int V, int COL>
__device__ __forceinline__ void pull19(const float* __restrict__ src, const LbmParams& p, const Cell c,
                                       const int idx, float (&h)[Q][V]) {
    const int nx = p.nx, ny = p.ny, nz = p.nz;
    const size_t N = (size_t)p.cells;
    const bool xlo = c.i == 0, xhi = c.i == nx - 1;
    const bool ylo = c.j == 0, yhi = c.j == ny - 1;
    const bool zlo = c.k == 0, zhi = c.k == nz - 1;
    // neighbour offsets with periodic wrap (a wall axis bounces / closes instead, decided below)
    const int dxm = xlo ? nx - 1 : -1, dxp = xhi ? 1 - nx : 1;
    const int dym = (ylo ? ny - 1 : -1) * nx, dyp = (yhi ? 1 - ny : 1) * nx;
    const int dzm = (zlo ? nz - 1 : -1) * nx * ny, dzp = (zhi ? 1 - nz : 1) * nx * ny;
    const bool bxlo = p.wall[0] == PLB_WALL_BB && xlo, bxhi = p.wall[0] == PLB_WALL_BB && xhi;
    const bool bylo = p.wall[1] == PLB_WALL_BB && ylo, byhi = p.wall[1] == PLB_WALL_BB && yhi;
    const bool bzlo = p.wall[2] == PLB_WALL_BB && zlo, bzhi = p.wall[2] == PLB_WALL_BB && zhi;
    // on-site velocity wall (at most one axis): face of this cell, 0 = none, +1 = low, -1 = high
    const int hx = p.wall[0] == PLB_WALL_HH ? (xlo ? 1 : (xhi ? -1 : 0)) : 0;
    const int hy = p.wall[1] == PLB_WALL_HH ? (ylo ? 1 : (yhi ? -1 : 0)) : 0;
    const int hz = p.wall[2] == PLB_WALL_HH ? (zlo ? 1 : (zhi ? -1 : 0)) : 0;
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
        // on-site wall: x - c_d lies beyond the face -> "undetermined" (L217), closed below
        const bool undetermined = (cx != 0 && cx == hx) || (cy != 0 && cy == hy) || (cz != 0 && cz == hz);
        if (undetermined) h[d][COL] = 0.f;
        else if (b) h[d][COL] = __ldg(src + (size_t)OPP(d) * N + idx) + corr;
        else        h[d][COL] = __ldg(src + (size_t)d * N + (idx + off));
    }
    if (hx) hecht_harting_close<0, V, COL>(h, hx, p.uw[0][hx < 0]);
    if (hy) hecht_harting_close<1, V, COL>(h, hy, p.uw[1][hy < 0]);
    if (hz) hecht_harting_close<2, V, COL>(h, hz, p.uw[2][hz < 0]);
}

// The same pull for a cell whose 18 neighbours all lie inside the grid (no wrap, no wall): the
// source offsets are compile-time multiples of the strides.
template <int V, int COL>
__device__ __forceinline__ void pull19_interior(const float* __restrict__ src, const size_t N, const int idx,
                                                const int sy, const int sz, float (&h)[Q][V]) {
#pragma unroll
    for (int d = 0; d < Q; ++d)
        h[d][COL] = __ldg(src + (size_t)d * N + (idx - CX(d) - CY(d) * sy - CZ(d) * sz));
}

// delta rho = sum h_d, j = sum c_d h_d (Eq. 17-18; sum_d w_d c_d = 0 so the shift drops out of j)
template <int V, int COL>
__device__ __forceinline__ void moments(const float (&h)[Q][V], float& drho, float& jx, float& jy, float& jz) {
    // pairwise sums keep the fp32 rounding small and symmetric
    const float a01p = h[0][COL] + h[1][COL], a23p = h[2][COL] + h[3][COL], a45p = h[4][COL] + h[5][COL];
    const float s6 = (h[6][COL] + h[11][COL]) + (h[7][COL] + h[10][COL]);      // xy diagonals
    const float s8 = (h[8][COL] + h[13][COL]) + (h[9][COL] + h[12][COL]);      // xz diagonals
    const float s14 = (h[14][COL] + h[17][COL]) + (h[15][COL] + h[16][COL]);   // yz diagonals
    drho = ((a01p + a23p) + (a45p + h[18][COL])) + ((s6 + s8) + s14);
    const float d611 = h[6][COL] - h[11][COL], d710 = h[7][COL] - h[10][COL];
    const float d813 = h[8][COL] - h[13][COL], d912 = h[9][COL] - h[12][COL];
    const float d1417 = h[14][COL] - h[17][COL], d1516 = h[15][COL] - h[16][COL];
    jx = (h[0][COL] - h[1][COL]) + ((d611 + d710) + (d813 + d912));
    jy = (h[2][COL] - h[3][COL]) + ((d611 - d710) + (d1417 + d1516));
    jz = (h[4][COL] - h[5][COL]) + ((d813 - d912) + (d1417 - d1516));
}

// rho and v = (j + g/2)/rho (Eq. 17-18) of the streamed state at cell (i,j,k), as
// (vx, vy, vz, rho); g = nullptr: no force.
__device__ __forceinline__ float4 cell_macros(const float* __restrict__ src, const float4* __restrict__ g,
                                              const LbmParams& p, const Cell c) {
    const int idx = c.i + p.nx * (c.j + p.ny * c.k);
    float h[Q][1];
    pull19<1, 0>(src, p, c, idx, h);
    float drho, jx, jy, jz;
    moments<1, 0>(h, drho, jx, jy, jz);
    float4 g4 = make_float4(0.f, 0.f, 0.f, 0.f);
    if (g) g4 = __ldg(g + idx);
    const float rho = 1.0f + drho, inv = 1.0f / rho;
    return make_float4((jx + 0.5f * g4.x) * inv, (jy + 0.5f * g4.y) * inv, (jz + 0.5f * g4.z) * inv, rho);
}

// the same for an interior cell (see pull19_interior)
__device__ __forceinline__ float4 cell_macros_interior(const float* __restrict__ src, const float4* __restrict__ g,
                                                       const LbmParams& p, const int idx) {
    float h[Q][1];
    pull19_interior<1, 0>(src, (size_t)p.cells, idx, p.nx, p.nx * p.ny, h);
    float drho, jx, jy, jz;
    moments<1, 0>(h, drho, jx, jy, jz);
    float4 g4 = make_float4(0.f, 0.f, 0.f, 0.f);
    if (g) g4 = __ldg(g + idx);
    const float rho = 1.0f + drho, inv = 1.0f / rho;
    return make_float4((jx + 0.5f * g4.x) * inv, (jy + 0.5f * g4.y) * inv, (jz + 0.5f * g4.z) * inv, rho);
}

}  // namespace plb
