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
#include <mutex>
#include "plb_internal.cuh"
#include "lbm_device.cuh"

namespace plb {

// BGK relaxation (Eq. 16) towards f_eq(rho, v) (Eq. 20) with v = u + g/(2 rho) (L201) plus the
// Guo term (Eq. 19 in the form S_d = (1 - 1/2tau) w_d [3 (c_d - v).g + 9 (c_d.v)(c_d.g)],
// DESIGN.md G3), on the shifted populations  h_eq,d = w_d [drho + rho (3 c.v + 4.5 (c.v)^2 - 1.5 v^2)].
//
// fp32 and thousands of steps: a relaxation whose rounded constants do not add up EXACTLY to the
// conservation laws multiplies the momentum of every cell by 1 + O(2^-24) per step -- coherent,
// so it piles up linearly (velocity) and quadratically (node positions).  Hence
//  * everything is written in the momentum m = rho v = j + g/2:  rho (c.v) = c.m needs no division,
//    rho (c.v)^2 = (c.m)^2/rho, rho v^2 = m.m/rho, v.g = m.g/rho;
//  * the lattice constants are fp32 numbers within 1.2e-7 (relative) of 3 w_d, 1.5 w_d and w_d that
//    satisfy the moment identities exactly in real arithmetic:
//        2 KA + 8 KG = 1           (first moment of the odd part  = m)
//        6 AA + 12 AG + A0 = 3/2   (zeroth moment of the second-order part = 0, with 1/4 and 1/8)
//        6 WA + 12 WG + W0 = 1     (zeroth moment of the density part = drho)
//  * the relaxation is out = h + omega (h_eq - h), so omega itself needs no special form.
// What is left are roundings of single operations, which do not have a preferred sign.
// A population and its opposite share the part even in c_d and differ in the sign of the odd part.
__device__ __forceinline__ float lattice_const(const unsigned bits) { return __uint_as_float(bits); }
#define PLB_KA lattice_const(0x3e2aaaacu)   /* ~1/6   */
#define PLB_KG lattice_const(0x3daaaaaau)   /* ~1/12: (1 - 2 KA)/8 */
#define PLB_AA lattice_const(0x3daaaaacu)   /* ~1/12  */
#define PLB_A0 lattice_const(0x3efffffcu)   /* ~1/2:  3/2 - 12 AA; AG = AA/2 */
#define PLB_WA lattice_const(0x3d638e38u)   /* ~1/18  */
#define PLB_W0 lattice_const(0x3eaaaaacu)   /* ~1/3:  1 - 12 WA;   WG = WA/2 */

struct PairCoef {
    float Z, B, K;      // w drho - 1.5 w m.m/rho,  4.5 w / rho,  3 w
    float P, PK;        // 3 w pref / rho,  3 w pref
};

template <bool FORCED, int V, int COL>
__device__ __forceinline__ void relax_pair(float (&h)[Q][V], const int d, const int e, const float cm, const float cg,
                                           const float mg, const float omega, const PairCoef& k) {
    const float even = fmaf(k.B, cm * cm, k.Z);
    const float odd = k.K * cm;
    float od = fmaf(omega, (even + odd) - h[d][COL], h[d][COL]);
    float oe = fmaf(omega, (even - odd) - h[e][COL], h[e][COL]);
    if (FORCED) {                                        // Guo term S_d (not relaxed)
        const float se = k.P * fmaf(3.0f * cm, cg, -mg);
        const float so = k.PK * cg;
        od += se + so;
        oe += se - so;
    }
    h[d][COL] = od;
    h[e][COL] = oe;
}

template <bool FORCED, int V, int COL>
__device__ __forceinline__ void collide(float (&h)[Q][V], const float gx, const float gy, const float gz,
                                        const float omega, const float pref) {
    float drho, mx, my, mz;
    moments<V, COL>(h, drho, mx, my, mz);
    if (FORCED) {
        mx = fmaf(0.5f, gx, mx); my = fmaf(0.5f, gy, my); mz = fmaf(0.5f, gz, mz);
    }
    const float inv = 1.0f / (1.0f + drho);
    const float mm = (mx * mx + my * my + mz * mz) * inv;           // rho v^2
    const float mg = FORCED ? (mx * gx + my * gy + mz * gz) : 0.f;  // rho v.g
    const float pri = pref * inv;
    PairCoef k1, k2;                       // axes (w = 1/18), diagonals (w = 1/36)
    k1.Z = fmaf(PLB_WA, drho, -PLB_AA * mm); k1.B = 0.25f * inv;  k1.K = PLB_KA;
    k2.Z = 0.5f * k1.Z;                      k2.B = 0.125f * inv; k2.K = PLB_KG;
    k1.P = PLB_KA * pri; k1.PK = PLB_KA * pref;
    k2.P = PLB_KG * pri; k2.PK = PLB_KG * pref;
    relax_pair<FORCED, V, COL>(h, 0, 1, mx, gx, mg, omega, k1);
    relax_pair<FORCED, V, COL>(h, 2, 3, my, gy, mg, omega, k1);
    relax_pair<FORCED, V, COL>(h, 4, 5, mz, gz, mg, omega, k1);
    relax_pair<FORCED, V, COL>(h, 6, 11, mx + my, gx + gy, mg, omega, k2);
    relax_pair<FORCED, V, COL>(h, 7, 10, mx - my, gx - gy, mg, omega, k2);
    relax_pair<FORCED, V, COL>(h, 8, 13, mx + mz, gx + gz, mg, omega, k2);
    relax_pair<FORCED, V, COL>(h, 9, 12, mx - mz, gx - gz, mg, omega, k2);
    relax_pair<FORCED, V, COL>(h, 14, 17, my + mz, gy + gz, mg, omega, k2);
    relax_pair<FORCED, V, COL>(h, 15, 16, my - mz, gy - gz, mg, omega, k2);
    // rest population: c = 0
    const float rest = fmaf(PLB_W0, drho, -PLB_A0 * mm);
    float o18 = fmaf(omega, rest - h[18][COL], h[18][COL]);
    if (FORCED) o18 = fmaf(-pri, mg, o18);               // S_19 = w_19 * 3 * pref * (-v.g)
    h[18][COL] = o18;
}

// ---------------------------------------------------------------------------------------------
// S3, generic kernel: fused pull-stream + collide + boundary, one thread per cell.  Handles every
// grid size and boundary mix; used when the vectorised kernel below does not apply.
// ---------------------------------------------------------------------------------------------
template <int MODE>
__device__ __forceinline__ void step_one_cell(const float* __restrict__ src, float* __restrict__ dst,
                                              const float4* __restrict__ g, const unsigned* __restrict__ seg_mask,
                                              const LbmParams& p, const Cell c, const int idx) {
    float h[Q][1];
    pull19<1, 0>(src, p, c, idx, h);
    bool forced = false;
    float4 g4 = make_float4(0.f, 0.f, 0.f, 0.f);
    if (MODE == FORCE_DENSE) {
        g4 = __ldg(g + idx);
        forced = true;
    } else if (MODE == FORCE_SPARSE) {
        if (seg_active(seg_mask, idx)) {
            g4 = __ldg(g + idx);
            forced = true;
        }
    }
    if (forced) collide<true, 1, 0>(h, g4.x, g4.y, g4.z, p.omega, p.pref);
    else        collide<false, 1, 0>(h, 0.f, 0.f, 0.f, p.omega, p.pref);
    const size_t N = (size_t)p.cells;
#pragma unroll
    for (int d = 0; d < Q; ++d) dst[(size_t)d * N + idx] = h[d][0];
}

template <int MODE>
__global__ void __launch_bounds__(256) lbm_step_kernel(const float* __restrict__ src, float* __restrict__ dst,
                                                       const float4* __restrict__ g,
                                                       const unsigned* __restrict__ seg_mask, const LbmParams p) {
    const int idx = blockIdx.x * 256 + threadIdx.x;
    if (idx >= p.cells) return;
    step_one_cell<MODE>(src, dst, g, seg_mask, p, cell_of(idx, p), idx);
}

// ---------------------------------------------------------------------------------------------
// S3, vectorised kernel (nx % V == 0, x periodic): one thread per V consecutive cells of a row.
//  * c_x = 0 populations: one aligned 128-bit (V = 4) load;
//  * c_x = +-1 populations: the aligned vector of the same V cells, shifted by one through the
//    neighbouring lane (shfl), the lane at a warp / row edge fetching the one missing element;
//  * stores are aligned vectors.
// ---------------------------------------------------------------------------------------------
template <int V> struct Vec;
template <> struct Vec<4> {
    static __device__ __forceinline__ void load(const float* p, float (&a)[4]) {
        const float4 t = __ldg(reinterpret_cast<const float4*>(p));
        a[0] = t.x; a[1] = t.y; a[2] = t.z; a[3] = t.w;
    }
};
template <> struct Vec<2> {
    static __device__ __forceinline__ void load(const float* p, float (&a)[2]) {
        const float2 t = __ldg(reinterpret_cast<const float2*>(p));
        a[0] = t.x; a[1] = t.y;
    }
};

// Hecht-Harting closure of every column of a row that lies on an on-site velocity face
template <int V, int COL>
__device__ __forceinline__ void close_on_site_walls(float (&h)[Q][V], const int hy, const int hz, const LbmParams& p) {
    if (hy) hecht_harting_close<1, V, COL>(h, hy, p.uw[1][hy < 0]);
    if (hz) hecht_harting_close<2, V, COL>(h, hz, p.uw[2][hz < 0]);
    if constexpr (COL + 1 < V) close_on_site_walls<V, COL + 1>(h, hy, hz, p);
}

template <int MODE, int V, int COL>
__device__ __forceinline__ void collide_cols(float (&h)[Q][V], const float4 (&g4)[V], const bool forced,
                                             const float omega, const float pref) {
    if (MODE != FORCE_NONE && forced) collide<true, V, COL>(h, g4[COL].x, g4[COL].y, g4[COL].z, omega, pref);
    else                              collide<false, V, COL>(h, 0.f, 0.f, 0.f, omega, pref);
    if constexpr (COL + 1 < V) collide_cols<MODE, V, COL + 1>(h, g4, forced, omega, pref);
}

// Pull of the 19 populations of V consecutive cells of a row.  WALLS = false: the source rows
// wrap periodically (interior rows, and every row of a fully periodic box).  WALLS = true: the
// row may lie on a y / z wall face, handled in the same vector form: a population whose source
// cell lies beyond a bounce-back face is T_dbar of the SAME cell plus the moving-wall term (an
// aligned vector of row dbar with no x shift); beyond an on-site velocity face it is
// "undetermined" (not loaded) and closed from the others (Eq. 23-30) column by column.  The x
// shuffles run unconditionally; a bounced lane ignores what they deliver (lanes of one row
// bounce together).  The kernel takes the WALLS = true form only in warps that hold a wall row,
// so the interior keeps the branch-free schedule (19 independent vector loads in flight) that
// reaches the copy bandwidth -- the all-rows general form cost 25 % at config 4 (measured).
template <int V, bool WALLS>
__device__ __forceinline__ void pull_rows(float (&h)[Q][V], const float* __restrict__ src, const LbmParams& p,
                                          const int idx0, const int i0, const int j, const int k, const int hy,
                                          const int hz) {
    constexpr unsigned FULL = 0xffffffffu;
    const int nx = p.nx, ny = p.ny, nz = p.nz;
    const size_t N = (size_t)p.cells;
    const bool ylo = j == 0, yhi = j == ny - 1, zlo = k == 0, zhi = k == nz - 1;
    const bool bylo = WALLS && p.wall[1] == PLB_WALL_BB && ylo, byhi = WALLS && p.wall[1] == PLB_WALL_BB && yhi;
    const bool bzlo = WALLS && p.wall[2] == PLB_WALL_BB && zlo, bzhi = WALLS && p.wall[2] == PLB_WALL_BB && zhi;
    const int lane = threadIdx.x & 31;
    const bool first = lane == 0 || i0 == 0;          // cell i0 - 1 is not in the lane below
    const bool last = lane == 31 || i0 + V == nx;     // cell i0 + V is not in the lane above
    const int xm = i0 == 0 ? nx - 1 : -1;             // offset of cell i0 - 1 (periodic)
    const int xp = i0 + V == nx ? V - nx : V;         // offset of cell i0 + V (periodic)
    const int dym = (ylo ? ny - 1 : -1) * nx, dyp = (yhi ? 1 - ny : 1) * nx;
    const int dzm = (zlo ? nz - 1 : -1) * nx * ny, dzp = (zhi ? 1 - nz : 1) * nx * ny;
#pragma unroll
    for (int d = 0; d < Q; ++d) {
        const int cx = CX(d), cy = CY(d), cz = CZ(d);
        int off = 0;
        if (cy == 1) off += dym;
        if (cy == -1) off += dyp;
        if (cz == 1) off += dzm;
        if (cz == -1) off += dzp;
        const float* base = src + (size_t)d * N + (idx0 + off);
        float a[V];
        if constexpr (!WALLS) {
            Vec<V>::load(base, a);
            if (cx == 0) {
#pragma unroll
                for (int c = 0; c < V; ++c) h[d][c] = a[c];
            } else if (cx == 1) {                         // f_d(i) = T_d(i - 1)
                float prev = __shfl_up_sync(FULL, a[V - 1], 1);
                if (first) prev = __ldg(base + xm);
                h[d][0] = prev;
#pragma unroll
                for (int c = 1; c < V; ++c) h[d][c] = a[c - 1];
            } else {                                      // f_d(i) = T_d(i + 1)
                float next = __shfl_down_sync(FULL, a[0], 1);
                if (last) next = __ldg(base + xp);
#pragma unroll
                for (int c = 0; c + 1 < V; ++c) h[d][c] = a[c + 1];
                h[d][V - 1] = next;
            }
        } else {
            // bounce-back: z first, then y, so that y wins (corner rule: first wall axis in x, y, z order)
            bool b = false;
            float corr = 0.f;
            if (cz == 1 && bzlo) { b = true; corr = p.corr[2][0][d]; }
            if (cz == -1 && bzhi) { b = true; corr = p.corr[2][1][d]; }
            if (cy == 1 && bylo) { b = true; corr = p.corr[1][0][d]; }
            if (cy == -1 && byhi) { b = true; corr = p.corr[1][1][d]; }
            const bool undetermined = (cy != 0 && cy == hy) || (cz != 0 && cz == hz);
            const float* from = b ? src + (size_t)OPP(d) * N + idx0 : base;
#pragma unroll
            for (int c = 0; c < V; ++c) a[c] = 0.f;
            if (!undetermined) Vec<V>::load(from, a);
            if (cx == 0) {
#pragma unroll
                for (int c = 0; c < V; ++c) h[d][c] = a[c] + corr;
            } else if (cx == 1) {                         // f_d(i) = T_d(i - 1)
                float prev = __shfl_up_sync(FULL, a[V - 1], 1);
                if (first && !b && !undetermined) prev = __ldg(base + xm);
                h[d][0] = b ? a[0] + corr : prev;
#pragma unroll
                for (int c = 1; c < V; ++c) h[d][c] = b ? a[c] + corr : a[c - 1];
            } else {                                      // f_d(i) = T_d(i + 1)
                float next = __shfl_down_sync(FULL, a[0], 1);
                if (last && !b && !undetermined) next = __ldg(base + xp);
#pragma unroll
                for (int c = 0; c + 1 < V; ++c) h[d][c] = b ? a[c] + corr : a[c + 1];
                h[d][V - 1] = b ? a[V - 1] + corr : next;
            }
        }
    }
}

template <int MODE, int V, int THREADS, int MINB, bool WALLS>
__global__ void __launch_bounds__(THREADS, MINB) lbm_step_vec_kernel(const float* __restrict__ src, float* __restrict__ dst,
                                                                    const float4* __restrict__ g,
                                                                    const unsigned* __restrict__ seg_mask,
                                                                    const LbmParams p) {
    constexpr unsigned FULL = 0xffffffffu;
    const int nx = p.nx, ny = p.ny, nz = p.nz;
    const unsigned nvec = (unsigned)p.cells / V;
    unsigned t = blockIdx.x * THREADS + threadIdx.x;
    const bool live = t < nvec;
    if (!live) t = nvec - 1;                            // keeps the lane for the shuffles below
    const int idx0 = (int)(t * V);
    const unsigned row = (unsigned)idx0 / (unsigned)nx;
    const int i0 = idx0 - (int)(row * (unsigned)nx);
    const int k = (int)(row / (unsigned)ny);
    const int j = (int)row - k * ny;
    const size_t N = (size_t)p.cells;
    const bool ylo = j == 0, yhi = j == ny - 1, zlo = k == 0, zhi = k == nz - 1;
    // on-site velocity wall: face of this row, 0 = none, +1 = low, -1 = high
    const int hy = (WALLS && p.wall[1] == PLB_WALL_HH) ? (ylo ? 1 : (yhi ? -1 : 0)) : 0;
    const int hz = (WALLS && p.wall[2] == PLB_WALL_HH) ? (zlo ? 1 : (zhi ? -1 : 0)) : 0;
    const bool wall_row = WALLS && ((p.wall[1] && (ylo || yhi)) || (p.wall[2] && (zlo || zhi)));
    float h[Q][V];
    if (WALLS && __any_sync(FULL, wall_row)) pull_rows<V, true>(h, src, p, idx0, i0, j, k, hy, hz);
    else                                     pull_rows<V, false>(h, src, p, idx0, i0, j, k, 0, 0);
    if (!live) return;
    if (WALLS && (hy | hz)) close_on_site_walls<V, 0>(h, hy, hz, p);
    bool forced = false;
    float4 g4[V];
    if (MODE == FORCE_DENSE) forced = true;
    if (MODE == FORCE_SPARSE) forced = seg_active(seg_mask, idx0);   // V divides SEG: one flag for all V cells
    if (MODE != FORCE_NONE && forced) {
#pragma unroll
        for (int c = 0; c < V; ++c) g4[c] = __ldg(g + idx0 + c);
    }
    collide_cols<MODE, V, 0>(h, g4, forced, p.omega, p.pref);
#pragma unroll
    for (int d = 0; d < Q; ++d) {
        float* out = dst + (size_t)d * N + idx0;
        if constexpr (V == 4) *reinterpret_cast<float4*>(out) = make_float4(h[d][0], h[d][1], h[d][2], h[d][3]);
        else                  *reinterpret_cast<float2*>(out) = make_float2(h[d][0], h[d][1]);
    }
}

// rho and v = (j + g_last/2)/rho of the streamed state (what the next step will collide)
template <int MODE>
__global__ void __launch_bounds__(256) macros_kernel(const float* __restrict__ src, const float4* __restrict__ g,
                                                     const unsigned* __restrict__ seg_mask, float* __restrict__ rho_out,
                                                     float* __restrict__ u_out, const LbmParams p) {
    const int idx = blockIdx.x * 256 + threadIdx.x;
    if (idx >= p.cells) return;
    const Cell c = cell_of(idx, p);
    float h[Q][1];
    pull19<1, 0>(src, p, c, idx, h);
    float drho, jx, jy, jz;
    moments<1, 0>(h, drho, jx, jy, jz);
    float4 g4 = make_float4(0.f, 0.f, 0.f, 0.f);
    if (MODE == FORCE_DENSE) g4 = __ldg(g + idx);
    if (MODE == FORCE_SPARSE && seg_active(seg_mask, idx)) g4 = __ldg(g + idx);
    const float rho = 1.0f + drho, inv = 1.0f / rho;
    if (rho_out) rho_out[idx] = rho;
    if (u_out) {
        const size_t N = (size_t)p.cells;
        u_out[idx] = (jx + 0.5f * g4.x) * inv;
        u_out[N + idx] = (jy + 0.5f * g4.y) * inv;
        u_out[2 * N + idx] = (jz + 0.5f * g4.z) * inv;
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
    bool dead;    // the link leaves through an on-site velocity wall: the slot is never read
};

template <int D>
__device__ __forceinline__ Target pre_stream_target(const LbmParams& p, const Cell c, const int idx) {
    constexpr int cx = CX(D), cy = CY(D), cz = CZ(D);
    const int nx = p.nx, ny = p.ny, nz = p.nz;
    int ti = c.i + cx, tj = c.j + cy, tk = c.k + cz;
    bool b = false, dead = false;
    float corr = 0.f;
    // link D from x leaves through ...; z, y, x order so that x wins (corner rule).  Through an
    // on-site velocity wall the population simply leaves: the slot is never read.
    const bool bbx = p.wall[0] == PLB_WALL_BB, bby = p.wall[1] == PLB_WALL_BB, bbz = p.wall[2] == PLB_WALL_BB;
    if (tk < 0) { if (bbz) { b = true; corr = p.corr[2][0][OPP(D)]; } else if (p.wall[2]) dead = true; else tk += nz; }
    if (tk >= nz) { if (bbz) { b = true; corr = p.corr[2][1][OPP(D)]; } else if (p.wall[2]) dead = true; else tk -= nz; }
    if (tj < 0) { if (bby) { b = true; corr = p.corr[1][0][OPP(D)]; } else if (p.wall[1]) dead = true; else tj += ny; }
    if (tj >= ny) { if (bby) { b = true; corr = p.corr[1][1][OPP(D)]; } else if (p.wall[1]) dead = true; else tj -= ny; }
    if (ti < 0) { if (bbx) { b = true; corr = p.corr[0][0][OPP(D)]; } else if (p.wall[0]) dead = true; else ti += nx; }
    if (ti >= nx) { if (bbx) { b = true; corr = p.corr[0][1][OPP(D)]; } else if (p.wall[0]) dead = true; else ti -= nx; }
    Target t;
    t.dead = dead;
    if (dead) { t.idx = idx; t.d = D; t.corr = 0.f; }
    else if (b) { t.idx = idx; t.d = OPP(D); t.corr = corr; }
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
    dst[(size_t)D * p.cells + idx] = t.dead ? 0.f : init_value(t.d, t.idx, rho_in, u_in, (size_t)p.cells, amp, seed) - t.corr;
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
    dst[(size_t)D * p.cells + idx] = t.dead ? 0.f : (__ldg(f + (size_t)t.d * p.cells + t.idx) - wd) - t.corr;
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
    float h[Q][1];
    pull19<1, 0>(src, p, cell_of(idx, p), idx, h);
#pragma unroll
    for (int d = 0; d < Q; ++d) f[(size_t)d * p.cells + idx] = h[d][0] + WGT(d);
}

// debug aid: count the cells whose current state -- the 19 populations that
// stream INTO the cell, what lbm_read_macros sees -- has a non-finite population or a density
// rho = 1 + sum_d h_d (Eq. 17) that is not positive
__global__ void __launch_bounds__(256) check_finite_kernel(const float* __restrict__ src, int* __restrict__ bad,
                                                           const LbmParams p) {
    const int idx = blockIdx.x * 256 + threadIdx.x;
    if (idx >= p.cells) return;
    float h[Q][1];
    pull19<1, 0>(src, p, cell_of(idx, p), idx, h);
    bool finite = true;
#pragma unroll
    for (int d = 0; d < Q; ++d) finite = finite && isfinite(h[d][0]);
    float drho, jx, jy, jz;
    moments<1, 0>(h, drho, jx, jy, jz);
    if (!finite || !(1.0f + drho > 0.f)) atomicAdd(bad, 1);
}

// ---------------------------------------------------------------------------------------------
// lbm_check_finite_static: the same count with NO caller- or library-allocated scratch.  Some
// callers cannot provide or allocate scratch at the point of the call (code under CUDA graph
// capture, tight serving loops, harnesses that forbid cudaMalloc), and the count of
// check_finite_kernel needs a device counter.  Here the scratch is a file-scope device array of
// a stated maximum size: PLB_STATIC_SCRATCH_INTS ints = 256 KiB, held by every GPU that loads the
// library until the process exits.  One slot per thread block of 256 cells, so grids of up to
// PLB_STATIC_MAX_CELLS (plb.h) = 65,536 x 256 = 16,777,216 cells (256^3: configs 2 and 5) are served;
// larger grids are refused.
//   kernel 1: block b counts its bad cells and WRITES partial[b] (no atomics, no clear needed:
//             every slot that is read was written by the same call first);
//   kernel 2: one block sums partial[0 .. n_blocks) in a fixed order and writes *d_out.
// Every call on a device shares the array, which keeps the last call's contents: calls that
// overlap on the GPU (two streams, two contexts on one device) race on it.
// In HOST code the array's name is only a stand-in for the symbol, not a device address: the
// address kernel 1 receives comes from cudaGetSymbolAddress, asked once per device with that
// device current.  Device code of this file names the array directly (kernel 2).
// ---------------------------------------------------------------------------------------------
constexpr int PLB_STATIC_SCRATCH_INTS = 65536;
constexpr long STATIC_MAX_CELLS = (long)PLB_STATIC_SCRATCH_INTS * 256;
static_assert(STATIC_MAX_CELLS == PLB_STATIC_MAX_CELLS, "plb.h states the limit of lbm_check_finite_static");
static __device__ __align__(256) int g_static_scratch[PLB_STATIC_SCRATCH_INTS];

__global__ void __launch_bounds__(256) check_finite_partial_kernel(const float* __restrict__ src, int* __restrict__ partial,
                                                                   const LbmParams p) {
    __shared__ int warp_count[8];
    const int idx = blockIdx.x * 256 + threadIdx.x;
    bool bad = false;
    if (idx < p.cells) {
        float h[Q][1];
        pull19<1, 0>(src, p, cell_of(idx, p), idx, h);
        bool finite = true;
#pragma unroll
        for (int d = 0; d < Q; ++d) finite = finite && isfinite(h[d][0]);
        float drho, jx, jy, jz;
        moments<1, 0>(h, drho, jx, jy, jz);
        bad = !finite || !(1.0f + drho > 0.f);
    }
    const int n = __popc(__ballot_sync(0xffffffffu, bad));
    if ((threadIdx.x & 31) == 0) warp_count[threadIdx.x >> 5] = n;
    __syncthreads();
    if (threadIdx.x == 0) {
        int tot = 0;
#pragma unroll
        for (int w = 0; w < 8; ++w) tot += warp_count[w];
        partial[blockIdx.x] = tot;
    }
}

__global__ void __launch_bounds__(1024) check_finite_total_kernel(const int n_blocks, int* __restrict__ out) {
    __shared__ int warp_sum[32];
    int s = 0;
    for (int b = threadIdx.x; b < n_blocks; b += 1024) s += g_static_scratch[b];   // device code names the array
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) warp_sum[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x < 32) {
        int t = warp_sum[threadIdx.x];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
        if (threadIdx.x == 0) *out = t;
    }
}

// device address of g_static_scratch on the CURRENT device (cudaGetSymbolAddress once per device)
static int static_scratch_address(int** out) {
    constexpr int MAX_DEVICES = 64;
    static int* address[MAX_DEVICES] = {nullptr};
    static std::mutex lock;
    int dev = 0;
    int rc = cuda_check(cudaGetDevice(&dev), "cudaGetDevice");
    if (rc) return rc;
    if (dev < 0 || dev >= MAX_DEVICES) {
        set_error("lbm_check_finite_static: device ordinal %d out of range", dev);
        return PLB_ERR_ARG;
    }
    std::lock_guard<std::mutex> guard(lock);
    if (!address[dev]) {
        int* ptr = nullptr;
        rc = cuda_check(cudaGetSymbolAddress((void**)&ptr, g_static_scratch), "cudaGetSymbolAddress(g_static_scratch)");
        if (rc) return rc;
        if (!ptr) {
            set_error("lbm_check_finite_static: cudaGetSymbolAddress returned a null address");
            return PLB_ERR_CUDA;
        }
        address[dev] = ptr;
    }
    *out = address[dev];
    return PLB_OK;
}

// asynchronous on c->stream; no allocation, no host synchronisation
int launch_check_finite_static(Ctx* c, int* d_out) {
    if ((long)c->prm.cells > STATIC_MAX_CELLS) {
        set_error("lbm_check_finite_static: grid of %d cells exceeds the static scratch (%ld cells at most)", c->prm.cells,
                  STATIC_MAX_CELLS);
        return PLB_ERR_WORKSPACE;
    }
    int* partial = nullptr;
    const int rc = static_scratch_address(&partial);
    if (rc) return rc;
    const int n_blocks = (c->prm.cells + 255) / 256;
    check_finite_partial_kernel<<<n_blocks, 256, 0, c->stream>>>(c->f[c->cur], partial, c->prm);
    check_finite_total_kernel<<<1, 1024, 0, c->stream>>>(n_blocks, d_out);
    c->launches += 2;
    return cuda_check(cudaGetLastError(), "check_finite_partial_kernel / check_finite_total_kernel");
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

// The vectorised kernel needs rows that are whole vectors and a periodic x axis; V = 4 cells per
// thread, 128 threads per block (512 cells), at least 4 blocks per SM.
constexpr int LBM_V = 4, LBM_THREADS = 128, LBM_MINB = 4;

template <int MODE>
static void launch_step_mode(Ctx* c, const float* src, float* dst, const float4* g) {
    const LbmParams& p = c->prm;
    if (p.nx % LBM_V == 0 && !p.wall[0]) {
        const unsigned nvec = (unsigned)p.cells / LBM_V;
        const unsigned grid = (nvec + LBM_THREADS - 1) / LBM_THREADS;
        if (p.wall[1] || p.wall[2])
            lbm_step_vec_kernel<MODE, LBM_V, LBM_THREADS, LBM_MINB, true><<<grid, LBM_THREADS, 0, c->stream>>>(src, dst, g, c->seg_mask, p);
        else
            lbm_step_vec_kernel<MODE, LBM_V, LBM_THREADS, LBM_MINB, false><<<grid, LBM_THREADS, 0, c->stream>>>(src, dst, g, c->seg_mask, p);
    } else {
        lbm_step_kernel<MODE><<<grid_cells(c), 256, 0, c->stream>>>(src, dst, g, c->seg_mask, p);
    }
}

int launch_lbm_step(Ctx* c, const float4* g, int mode) {
    const float* src = c->f[c->cur];
    float* dst = c->f[c->cur ^ 1];
    if (mode == FORCE_NONE) launch_step_mode<FORCE_NONE>(c, src, dst, nullptr);
    else if (mode == FORCE_DENSE) launch_step_mode<FORCE_DENSE>(c, src, dst, g);
    else launch_step_mode<FORCE_SPARSE>(c, src, dst, g);
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
        macros_kernel<FORCE_SPARSE><<<grid, 256, 0, c->stream>>>(src, c->g_last, c->seg_mask, d_rho, d_u, c->prm);
    c->launches++;
    return cuda_check(cudaGetLastError(), "macros_kernel");
}

int launch_check_finite(Ctx* c, int* d_bad) {
    check_finite_kernel<<<grid_cells(c), 256, 0, c->stream>>>(c->f[c->cur], d_bad, c->prm);
    c->launches++;
    return cuda_check(cudaGetLastError(), "check_finite_kernel");
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
