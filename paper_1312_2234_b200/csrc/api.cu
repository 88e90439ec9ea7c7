// api.cu -- the C-ABI of libplb (include/plb.h): argument checks, workspace carving, call-order
// bookkeeping.  Every step of the path runs in the kernels of lbm.cu / ib.cu.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include "plb_internal.cuh"

namespace plb {

static thread_local char g_err[512] = "";

void set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

int cuda_check(cudaError_t e, const char* what) {
    if (e == cudaSuccess) return PLB_OK;
    set_error("%s: %s", what, cudaGetErrorString(e));
    return PLB_ERR_CUDA;
}

static size_t align_up(size_t v) { return (v + 255) & ~(size_t)255; }

struct Carve {
    char* base;
    size_t off;
    template <typename T>
    T* take(size_t count) {
        T* p = reinterpret_cast<T*>(base + off);
        off += align_up(count * sizeof(T));
        return p;
    }
};

// lays out the workspace; with base == nullptr it only measures
static size_t carve(Ctx* c, char* base, long cells, long n_segs, long max_nodes, long max_edges) {
    Carve w{base, 0};
    float* f0 = w.take<float>((size_t)Q * cells);
    float* f1 = w.take<float>((size_t)Q * cells);
    unsigned* seg_mask = w.take<unsigned>((size_t)(n_segs + 31) / 32);
    int* counters = w.take<int>(64);
    int* seg_list = w.take<int>((size_t)n_segs);
    float4* vfield = w.take<float4>((size_t)n_segs * SEG);
    double* X0 = w.take<double>((size_t)max_nodes);
    double* X1 = w.take<double>((size_t)max_nodes);
    double* X2 = w.take<double>((size_t)max_nodes);
    float4* F = w.take<float4>((size_t)max_nodes);
    float4* U = w.take<float4>((size_t)max_nodes);
    double* stage = w.take<double>((size_t)3 * max_nodes);
    int* csr_off = w.take<int>((size_t)2 * max_nodes + 2);
    int2* csr_ent = w.take<int2>((size_t)2 * max_edges);
    int2* ranges = w.take<int2>((size_t)max_nodes);
    int* orig = w.take<int>((size_t)max_nodes);
    const long box_cap = max_nodes / 16 + 4096;
    int* range_box = w.take<int>((size_t)8 * box_cap);
    // a closed genus-0 triangulated surface of N nodes has 2N - 4 triangles and at least 4 nodes
    int4* tris = w.take<int4>((size_t)2 * max_nodes);
    float* tri_S0 = w.take<float>((size_t)2 * max_nodes);
    MeshConstraint* cons = w.take<MeshConstraint>((size_t)max_nodes / 4 + 1);
    if (c) {
        c->tris = tris; c->tri_S0 = tri_S0; c->cons = cons;
        c->cap_tris = 2 * max_nodes; c->cap_cons = max_nodes / 4 + 1;
        c->f[0] = f0; c->f[1] = f1;
        c->seg_mask = seg_mask; c->counters = counters; c->seg_list = seg_list; c->vfield = vfield;
        c->X[0] = X0; c->X[1] = X1; c->X[2] = X2; c->F = F; c->U = U; c->stage = stage;
        c->csr_off = csr_off; c->csr_ent = csr_ent; c->ranges = ranges; c->orig = orig;
        c->range_box = range_box; c->box_cap = (int)box_cap;
    }
    return w.off;
}

// Order of the nodes of one mesh along the Morton (Z-order) curve of its shape: 10 bits per axis
// over the cube that bounds the mesh, ties broken by the caller's index.  ord[j] = caller's local
// index of the j-th stored node.
static unsigned spread_bits10(unsigned v) {
    v &= 0x3ffu;
    v = (v | (v << 16)) & 0x030000ffu;
    v = (v | (v << 8)) & 0x0300f00fu;
    v = (v | (v << 4)) & 0x030c30c3u;
    v = (v | (v << 2)) & 0x09249249u;
    return v;
}
static std::vector<int> morton_order(const double* xyz, int n) {
    double lo[3] = {xyz[0], xyz[1], xyz[2]}, hi[3] = {xyz[0], xyz[1], xyz[2]};
    for (int m = 1; m < n; ++m)
        for (int d = 0; d < 3; ++d) {
            lo[d] = xyz[3 * m + d] < lo[d] ? xyz[3 * m + d] : lo[d];
            hi[d] = xyz[3 * m + d] > hi[d] ? xyz[3 * m + d] : hi[d];
        }
    double ext = 0.0;
    for (int d = 0; d < 3; ++d) ext = hi[d] - lo[d] > ext ? hi[d] - lo[d] : ext;
    const double scale = (ext > 0.0 && std::isfinite(ext)) ? 1023.0 / ext : 0.0;
    std::vector<unsigned> code((size_t)n);
    for (int m = 0; m < n; ++m) {
        unsigned q[3];
        for (int d = 0; d < 3; ++d) {
            const double t = (xyz[3 * m + d] - lo[d]) * scale;
            q[d] = t >= 0.0 && t <= 1023.0 ? (unsigned)t : 0u;
        }
        code[m] = spread_bits10(q[0]) | (spread_bits10(q[1]) << 1) | (spread_bits10(q[2]) << 2);
    }
    std::vector<int> ord((size_t)n);
    for (int m = 0; m < n; ++m) ord[m] = m;
    std::sort(ord.begin(), ord.end(), [&](int a, int b) { return code[a] != code[b] ? code[a] < code[b] : a < b; });
    return ord;
}

static int __float_as_int_host(float f) {
    int i;
    memcpy(&i, &f, sizeof(i));
    return i;
}

static int check_grid(const plb_grid* g, long* cells) {
    if (!g || g->nx < 1 || g->ny < 1 || g->nz < 1) {
        set_error("invalid grid");
        return PLB_ERR_ARG;
    }
    const long long n = (long long)g->nx * g->ny * g->nz;
    if (n >= (1LL << 31) - 256) {
        set_error("grid too large: %lld cells (limit 2^31)", n);
        return PLB_ERR_ARG;
    }
    *cells = (long)n;
    return PLB_OK;
}

static int sync_status(Ctx* c) {
    int rc = cuda_check(cudaStreamSynchronize(c->stream), "cudaStreamSynchronize");
    if (rc) return rc;
    int h[2] = {0, 0};
    rc = cuda_check(cudaMemcpy(h, c->counters, sizeof(h), cudaMemcpyDeviceToHost), "read status");
    if (rc) return rc;
    if (h[1] & STATUS_ZERO_EDGE) {
        set_error("a mesh edge has zero length");
        return PLB_ERR_ARG;
    }
    if (h[1] & STATUS_ADH_BAD_SITE) {
        set_error("ib_write_bonds: a bond names a site outside a non-periodic tangential axis");
        return PLB_ERR_ARG;
    }
    if (h[1] & STATUS_NODE_LEFT) {
        set_error("a node left the channel through a wall axis");
        return PLB_ERR_NODE_LEFT;
    }
    return PLB_OK;
}

}  // namespace plb

// host-side geometry of one unstressed mesh: S_0 per triangle, S0_tot, V_0 (plain fp64; set-up only)
namespace plb {
void reference_area_volume(const double* x, int n_tris, const int* tris, float* S0, double* S0_tot, double* V0) {
    double S = 0, V6 = 0;
    for (int t = 0; t < n_tris; ++t) {
        const double* a = x + 3 * tris[3 * t];
        const double* b = x + 3 * tris[3 * t + 1];
        const double* c = x + 3 * tris[3 * t + 2];
        const double ab[3] = {b[0] - a[0], b[1] - a[1], b[2] - a[2]}, ac[3] = {c[0] - a[0], c[1] - a[1], c[2] - a[2]};
        const double n[3] = {ab[1] * ac[2] - ab[2] * ac[1], ab[2] * ac[0] - ab[0] * ac[2], ab[0] * ac[1] - ab[1] * ac[0]};
        const double s = 0.5 * sqrt(n[0] * n[0] + n[1] * n[1] + n[2] * n[2]);
        S0[t] = (float)s;
        S += s;
        // relative to the mesh's first node (V is translation invariant for a closed surface)
        const double* o = x;
        const double ra[3] = {a[0] - o[0], a[1] - o[1], a[2] - o[2]}, rb[3] = {b[0] - o[0], b[1] - o[1], b[2] - o[2]},
                     rc[3] = {c[0] - o[0], c[1] - o[1], c[2] - o[2]};
        V6 += ra[0] * (rb[1] * rc[2] - rb[2] * rc[1]) + ra[1] * (rb[2] * rc[0] - rb[0] * rc[2]) +
              ra[2] * (rb[0] * rc[1] - rb[1] * rc[0]);
    }
    *S0_tot = S;
    *V0 = V6 / 6.0;
}
}  // namespace plb

using namespace plb;

#define REQUIRE_CTX(ctx)                 \
    if (!(ctx)) {                        \
        set_error("null context");       \
        return PLB_ERR_ARG;              \
    }

extern "C" {

const char* plb_last_error(void) { return g_err; }

int lbm_workspace_bytes(const plb_grid* grid, long max_nodes, long max_edges, size_t* out_bytes) {
    long cells;
    int rc = check_grid(grid, &cells);
    if (rc) return rc;
    if (!out_bytes || max_nodes < 0 || max_edges < 0) {
        set_error("invalid capacity / null output");
        return PLB_ERR_ARG;
    }
    const long n_segs = (cells + SEG - 1) / SEG;
    *out_bytes = carve(nullptr, nullptr, cells, n_segs, max_nodes, max_edges);
    return PLB_OK;
}

int lbm_create(const plb_grid* grid, float tau, const plb_boundary* bnd, void* d_workspace, size_t workspace_bytes,
               long max_nodes, long max_edges, void* cuda_stream, plb_ctx** out) {
    long cells;
    int rc = check_grid(grid, &cells);
    if (rc) return rc;
    if (!out || !bnd || !d_workspace || !(tau > 0.5f) || max_nodes < 0 || max_edges < 0) {
        set_error("lbm_create: invalid argument (tau must exceed 1/2)");
        return PLB_ERR_ARG;
    }
    if (((uintptr_t)d_workspace & 255) != 0) {
        set_error("lbm_create: workspace must be 256-byte aligned");
        return PLB_ERR_ARG;
    }
    for (int a = 0; a < 3; ++a)
        if (bnd->kind[a] != PLB_PERIODIC && bnd->kind[a] != PLB_WALL_BB && bnd->kind[a] != PLB_WALL_HH) {
            set_error("lbm_create: invalid boundary kind on axis %d", a);
            return PLB_ERR_ARG;
        }
    for (int a = 0; a < 3; ++a)
        if (bnd->kind[a] == PLB_WALL_HH) {
            const int na = a == 0 ? grid->nx : (a == 1 ? grid->ny : grid->nz);
            if (na < 2 || bnd->kind[(a + 1) % 3] != PLB_PERIODIC || bnd->kind[(a + 2) % 3] != PLB_PERIODIC) {
                set_error("lbm_create: PLB_WALL_HH on axis %d needs n >= 2 and the other two axes periodic", a);
                return PLB_ERR_ARG;
            }
        }
    const long n_segs = (cells + SEG - 1) / SEG;
    const size_t need = carve(nullptr, nullptr, cells, n_segs, max_nodes, max_edges);
    if (workspace_bytes < need) {
        set_error("lbm_create: workspace of %zu bytes is smaller than the %zu needed", workspace_bytes, need);
        return PLB_ERR_WORKSPACE;
    }
    int dev = 0, sms = 0;
    rc = cuda_check(cudaGetDevice(&dev), "cudaGetDevice");
    if (rc) return rc;
    rc = cuda_check(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev), "cudaDeviceGetAttribute");
    if (rc) return rc;

    plb_ctx* c = new (std::nothrow) plb_ctx();
    if (!c) {
        set_error("out of host memory");
        return PLB_ERR_ARG;
    }
    c->grid = *grid;
    c->tau = tau;
    c->bnd = *bnd;
    c->stream = (cudaStream_t)cuda_stream;
    c->n_segs = n_segs;
    c->cur = 0;
    c->cap_nodes = max_nodes; c->cap_edges = max_edges; c->n_nodes = 0; c->n_edges = 0;
    c->g_last = nullptr; c->g_last_mode = FORCE_NONE; c->spread_target = nullptr;
    c->spread_current = false; c->listed_all = false; c->forces_valid = false; c->populated = false;
    c->launches = 0;
    c->n_ranges = 0;
    c->n_csr_off = 0; c->n_csr_ent = 0;
    c->n_tris = 0; c->n_cons = 0;
    c->adh_on = false; c->n_rec = 0;
    c->list_parity = 0;
    c->tile_cap = 512;
    c->spread_cap = 1024;
    c->spread_mode = PLB_SPREAD_AUTO;
    c->interp_form = PLB_INTERP_AUTO;
    if (const char* e = getenv("PLB_INTERP")) {                         // measurement knob
        if (!strcmp(e, "direct")) c->interp_form = PLB_INTERP_DIRECT;
        if (!strcmp(e, "tile")) c->interp_form = PLB_INTERP_TILE;
        if (!strcmp(e, "pull")) c->interp_form = PLB_INTERP_PULL;
    }
    c->range_nodes = 0;
    if (const char* e = getenv("PLB_RANGE_NODES")) c->range_nodes = atoi(e);   // measurement knob: nodes per IB block
    c->tile_nodes = 0.0; c->tile_cells = 0.0; c->tile_density = 0.0;
    c->sm_count = sms;
    c->mesh_node_off.push_back(0);
    c->mesh_edge_off.push_back(0);
    carve(c, (char*)d_workspace, cells, n_segs, max_nodes, max_edges);
    if (const char* e = getenv("PLB_BOX_CAP")) {                        // test knob: ranges whose box the spread stores
        const int v = atoi(e);
        if (v >= 0 && v < c->box_cap) c->box_cap = v;
    }

    LbmParams& p = c->prm;
    p.nx = grid->nx; p.ny = grid->ny; p.nz = grid->nz; p.cells = (int)cells;
    p.omega = 1.0f / tau;
    p.pref = 1.0f - 0.5f / tau;
    for (int a = 0; a < 3; ++a) {
        p.wall[a] = bnd->kind[a];
        for (int d = 0; d < 3; ++d) {
            p.uw[a][0][d] = bnd->u_lo[a][d];
            p.uw[a][1][d] = bnd->u_hi[a][d];
        }
        for (int d = 0; d < Q; ++d) {
            const double w = d < 6 ? 1.0 / 18.0 : (d < 18 ? 1.0 / 36.0 : 1.0 / 3.0);
            const double lo = CX(d) * (double)bnd->u_lo[a][0] + CY(d) * (double)bnd->u_lo[a][1] + CZ(d) * (double)bnd->u_lo[a][2];
            const double hi = CX(d) * (double)bnd->u_hi[a][0] + CY(d) * (double)bnd->u_hi[a][1] + CZ(d) * (double)bnd->u_hi[a][2];
            p.corr[a][0][d] = (float)(6.0 * w * lo);
            p.corr[a][1][d] = (float)(6.0 * w * hi);
        }
    }
    rc = cuda_check(cudaMemsetAsync(c->seg_mask, 0, (size_t)((n_segs + 31) / 32) * sizeof(unsigned), c->stream), "clear segment mask");
    if (!rc) rc = cuda_check(cudaMemsetAsync(c->counters, 0, 64 * sizeof(int), c->stream), "clear counters");
    // the velocity field only ever holds what segment_macros_kernel wrote; start it from finite values
    if (!rc) rc = cuda_check(cudaMemsetAsync(c->vfield, 0, (size_t)n_segs * SEG * sizeof(float4), c->stream), "clear velocity field");
    if (rc) {
        delete c;
        return rc;
    }
    *out = c;
    return PLB_OK;
}

int lbm_destroy(plb_ctx* ctx) {
    REQUIRE_CTX(ctx);
    cudaStreamSynchronize(ctx->stream);
    delete ctx;
    return PLB_OK;
}

int lbm_set_equilibrium(plb_ctx* ctx, const float* d_rho, const float* d_u, float noise_amp, unsigned long long seed) {
    REQUIRE_CTX(ctx);
    if (noise_amp < 0.f) {
        set_error("noise_amp must be >= 0");
        return PLB_ERR_ARG;
    }
    ctx->g_last = nullptr;
    ctx->g_last_mode = FORCE_NONE;
    ctx->populated = true;
    return launch_set_equilibrium(ctx, d_rho, d_u, noise_amp, seed);
}

int lbm_step(plb_ctx* ctx, const float* d_forcing) {
    REQUIRE_CTX(ctx);
    if (!ctx->populated) {
        set_error("lbm_step before lbm_set_equilibrium / lbm_write_populations");
        return PLB_ERR_ORDER;
    }
    int mode = FORCE_NONE;
    if (d_forcing) {
        if (((uintptr_t)d_forcing & 15) != 0) {
            set_error("forcing buffer must be 16-byte aligned (float4 per cell)");
            return PLB_ERR_ARG;
        }
        mode = ((const float4*)d_forcing == ctx->spread_target) ? FORCE_SPARSE : FORCE_DENSE;
    }
    const int rc = launch_lbm_step(ctx, (const float4*)d_forcing, mode);
    ctx->g_last = (const float4*)d_forcing;
    ctx->g_last_mode = mode;
    return rc;
}

int lbm_read_macros(plb_ctx* ctx, float* d_rho, float* d_u) {
    REQUIRE_CTX(ctx);
    if (!ctx->populated) {
        set_error("lbm_read_macros before the populations were set");
        return PLB_ERR_ORDER;
    }
    if (!d_rho && !d_u) return PLB_OK;
    return launch_read_macros(ctx, d_rho, d_u);
}

int lbm_read_populations(plb_ctx* ctx, float* d_f) {
    REQUIRE_CTX(ctx);
    if (!d_f || !ctx->populated) {
        set_error("lbm_read_populations: null output or populations not set");
        return d_f ? PLB_ERR_ORDER : PLB_ERR_ARG;
    }
    return launch_read_populations(ctx, d_f);
}

int lbm_write_populations(plb_ctx* ctx, const float* d_f) {
    REQUIRE_CTX(ctx);
    if (!d_f) {
        set_error("lbm_write_populations: null input");
        return PLB_ERR_ARG;
    }
    ctx->g_last = nullptr;
    ctx->g_last_mode = FORCE_NONE;
    ctx->populated = true;
    return launch_write_populations(ctx, d_f);
}

// ------------------------------------------------------------------------------------------------
int ib_add_meshes(plb_ctx* ctx, int n_meshes, int n_nodes, const double* h_xyz, int n_edges, const int* h_edges,
                  const float* h_rest, float k, int* out_first_mesh_id) {
    REQUIRE_CTX(ctx);
    if (n_meshes < 1 || n_nodes < 1 || !h_xyz || n_edges < 0 || (n_edges > 0 && !h_edges)) {
        set_error("ib_add_meshes: invalid argument");
        return PLB_ERR_ARG;
    }
    for (int e = 0; e < n_edges; ++e) {
        const int a = h_edges[2 * e], b = h_edges[2 * e + 1];
        if (a < 0 || a >= n_nodes || b < 0 || b >= n_nodes || a == b) {
            set_error("ib_add_meshes: edge %d = (%d, %d) is out of range or degenerate", e, a, b);
            return PLB_ERR_ARG;
        }
    }
    if (!h_rest && n_meshes > 1 && n_edges > 0) {
        // rest lengths = each mesh's own initial lengths: the meshes do not share one spring table
        for (int s = 0; s < n_meshes; ++s) {
            int id = 0;
            const int rc = ib_add_meshes(ctx, 1, n_nodes, h_xyz + (size_t)3 * s * n_nodes, n_edges, h_edges, nullptr, k, &id);
            if (rc) return rc;
            if (s == 0 && out_first_mesh_id) *out_first_mesh_id = id;
        }
        return PLB_OK;
    }
    const long add_nodes = (long)n_meshes * n_nodes, add_edges = (long)n_meshes * n_edges;
    if (ctx->n_nodes + add_nodes > ctx->cap_nodes || ctx->n_edges + add_edges > ctx->cap_edges) {
        set_error("ib_add_meshes: capacity exceeded (%ld/%ld nodes, %ld/%ld edges)", ctx->n_nodes + add_nodes,
                  ctx->cap_nodes, ctx->n_edges + add_edges, ctx->cap_edges);
        return PLB_ERR_WORKSPACE;
    }
    if (ctx->n_nodes + add_nodes >= (1L << 31)) {
        set_error("ib_add_meshes: more than 2^31 nodes");
        return PLB_ERR_ARG;
    }
    // Internal node order (hidden behind every call that names a node: ib_read/write_*, triangles,
    // receptors, the noise key): the nodes of a mesh are stored along the Morton curve of the first
    // mesh's shape.  The topology is fixed, so nodes that are consecutive in storage stay
    // neighbours on the surface however the mesh moves or deforms: a run of consecutive nodes is a
    // compact patch (small lattice tile, several blocks per mesh), and the two ends of an edge lie
    // close together in memory.
    const std::vector<int> ord = morton_order(h_xyz, n_nodes);           // ord[stored local] = caller's local
    std::vector<int> inv((size_t)n_nodes);
    for (int j = 0; j < n_nodes; ++j) inv[ord[j]] = j;
    // host-side marshalling: AoS -> SoA positions, mesh-local -> global edge indices
    std::vector<double> soa((size_t)3 * add_nodes);
    std::vector<int> og((size_t)add_nodes);
    for (int s = 0; s < n_meshes; ++s)
        for (int j = 0; j < n_nodes; ++j) {
            const long m = (long)s * n_nodes + j, src = (long)s * n_nodes + ord[j];
            for (int d = 0; d < 3; ++d) soa[(size_t)d * add_nodes + m] = h_xyz[3 * src + d];
            og[m] = (int)(ctx->n_nodes + src);
        }
    // Spring table of the topology (S1 is a gather: every node sums over its incident edges), in
    // stored local indices, ONE table for all meshes of the call: row i = the (neighbour, rest
    // length) pairs of node i, neighbours ascending.  A call that repeats the previous call's
    // topology, rest lengths and stiffness extends that group instead of adding a table.
    std::vector<float> rest((size_t)n_edges);
    for (int e = 0; e < n_edges; ++e) {
        if (h_rest) rest[e] = h_rest[e];
        else {
            const int a = h_edges[2 * e], b = h_edges[2 * e + 1];
            double s2 = 0;
            for (int d = 0; d < 3; ++d) s2 += (h_xyz[3 * b + d] - h_xyz[3 * a + d]) * (h_xyz[3 * b + d] - h_xyz[3 * a + d]);
            rest[e] = (float)sqrt(s2);
        }
    }
    bool extend = false;
    if (!ctx->groups.empty()) {
        const SpringGroupHost& last = ctx->group_src.back();
        extend = last.nn == n_nodes && last.k == k && (int)last.rest.size() == n_edges &&
                 std::equal(last.rest.begin(), last.rest.end(), rest.begin()) &&
                 std::equal(last.edges.begin(), last.edges.end(), h_edges);
    }
    std::vector<int> off;
    std::vector<int2> ent;
    if (!extend) {
        struct Half { int i, j; float L; };
        std::vector<Half> half((size_t)2 * n_edges);
        for (int e = 0; e < n_edges; ++e) {
            const int a = inv[h_edges[2 * e]], b = inv[h_edges[2 * e + 1]];
            half[2 * e] = Half{a, b, rest[e]};
            half[2 * e + 1] = Half{b, a, rest[e]};
        }
        std::stable_sort(half.begin(), half.end(), [](const Half& p, const Half& q) { return p.i != q.i ? p.i < q.i : p.j < q.j; });
        off.assign((size_t)n_nodes + 1, 0);
        ent.resize(half.size());
        for (size_t t = 0; t < half.size(); ++t) {
            off[half[t].i + 1]++;
            ent[t] = make_int2(half[t].j, __float_as_int_host(half[t].L));
        }
        for (int i = 0; i < n_nodes; ++i) off[i + 1] += off[i];
        for (int i = 0; i <= n_nodes; ++i) off[i] += (int)ctx->n_csr_ent;      // rows index the global entry array
    }
    // Node ranges of the IB thread blocks: a mesh, cut into runs of consecutive stored nodes (=
    // surface patches) so that the IB kernels get about two blocks per SM even when there are few
    // meshes (Eq. 33-34 are sums over nodes with no per-mesh structure), and never longer than
    // IB_RANGE_NODES.  Tile capacity: what the initial bounding boxes of the ranges ask for (two
    // cells of slack per axis for deformation).
    constexpr int IB_RANGE_NODES = 4096, IB_MIN_RANGE_NODES = 64;
    const long meshes_after = (long)ctx->mesh_node_off.size() - 1 + n_meshes;
    long parts = (2L * ctx->sm_count + meshes_after - 1) / meshes_after;
    if (parts > n_nodes / IB_MIN_RANGE_NODES) parts = n_nodes / IB_MIN_RANGE_NODES;
    if (ctx->range_nodes > 0) parts = (n_nodes + ctx->range_nodes - 1) / ctx->range_nodes;
    if (parts < (n_nodes + IB_RANGE_NODES - 1) / IB_RANGE_NODES) parts = (n_nodes + IB_RANGE_NODES - 1) / IB_RANGE_NODES;
    if (parts < 1) parts = 1;
    std::vector<int2> rg;
    int cap = ctx->tile_cap, scap = ctx->spread_cap;
    for (int s = 0; s < n_meshes; ++s) {
        const long noff = ctx->n_nodes + (long)s * n_nodes;
        const double* x = h_xyz + (size_t)3 * s * n_nodes;
        for (long part = 0; part < parts; ++part) {
            const int a = (int)((long)n_nodes * part / parts), b = (int)((long)n_nodes * (part + 1) / parts);
            if (b <= a) continue;
            rg.push_back(make_int2((int)(noff + a), (int)(noff + b)));
            double vol = 1.0, box = 1.0;
            int ext[3];
            for (int d = 0; d < 3; ++d) {
                double lo = floor(x[3 * ord[a] + d]), hi = lo;
                for (int m = a + 1; m < b; ++m) {
                    const double f = floor(x[3 * ord[m] + d]);
                    lo = f < lo ? f : lo;
                    hi = f > hi ? f : hi;
                }
                vol *= hi - lo + 4.0 + 2.0;
                box *= hi - lo + 4.0;
                ext[d] = hi - lo < 1e6 ? (int)(hi - lo) + 6 : 1 << 20;
            }
            // A mesh may turn (a flipping platelet).  The spread tile is sized for the cube of the
            // largest extent when that fits; the interpolation tile, whose kernel wants the L1 cache
            // that shared memory takes away (measured: 105 KB instead of 78 KB per block costs 45 %),
            // for the initial box, but for at least min(cube, 4352 cells).
            ctx->tile_nodes += (double)(b - a);
            ctx->tile_cells += box;
            const int emax = ext[0] > ext[1] ? (ext[0] > ext[2] ? ext[0] : ext[2]) : (ext[1] > ext[2] ? ext[1] : ext[2]);
            const double cube = (double)emax * emax * emax;
            if (vol <= (double)ib_max_tile_cap()) {
                double want = vol;
                const double allowance = cube < 4352.0 ? cube : 4352.0;
                if (want < allowance) want = allowance;
                if ((int)want > cap) cap = (int)want;
                int padded = tile_plane_pitch(tile_row_pitch(emax), emax) * emax;
                if (padded > ib_max_spread_cap()) padded = tile_plane_pitch(tile_row_pitch(ext[0]), ext[1]) * ext[2];
                if (padded <= ib_max_spread_cap() && padded > scap) scap = padded;
            }
        }
    }
    if (const char* e = getenv("PLB_TILE_CAP")) {                       // measurement knob: cells of the interpolation tile
        const int v = atoi(e);
        if (v >= 64 && v <= ib_max_tile_cap()) cap = v;
    }
    ctx->tile_cap = cap;
    ctx->spread_cap = scap;
    ctx->tile_density = ctx->tile_cells > 0.0 ? ctx->tile_nodes / ctx->tile_cells : 0.0;
    int rc = cuda_check(cudaMemcpyAsync(ctx->ranges + ctx->n_ranges, rg.data(), rg.size() * sizeof(int2),
                                        cudaMemcpyHostToDevice, ctx->stream), "upload node ranges");
    for (int d = 0; d < 3 && !rc; ++d)
        rc = cuda_check(cudaMemcpyAsync(ctx->X[d] + ctx->n_nodes, soa.data() + (size_t)d * add_nodes,
                                        (size_t)add_nodes * sizeof(double), cudaMemcpyHostToDevice, ctx->stream),
                        "upload node positions");
    if (!rc) rc = cuda_check(cudaMemcpyAsync(ctx->orig + ctx->n_nodes, og.data(), (size_t)add_nodes * sizeof(int),
                                             cudaMemcpyHostToDevice, ctx->stream), "upload node order");
    if (!rc) rc = cuda_check(cudaMemsetAsync(ctx->F + ctx->n_nodes, 0, (size_t)add_nodes * sizeof(float4), ctx->stream), "clear forces");
    if (!rc) rc = cuda_check(cudaMemsetAsync(ctx->U + ctx->n_nodes, 0, (size_t)add_nodes * sizeof(float4), ctx->stream), "clear node velocities");
    if (!rc && !extend) {
        rc = cuda_check(cudaMemcpyAsync(ctx->csr_off + ctx->n_csr_off, off.data(), off.size() * sizeof(int),
                                        cudaMemcpyHostToDevice, ctx->stream), "upload spring table rows");
        if (!rc && !ent.empty())
            rc = cuda_check(cudaMemcpyAsync(ctx->csr_ent + ctx->n_csr_ent, ent.data(), ent.size() * sizeof(int2),
                                            cudaMemcpyHostToDevice, ctx->stream), "upload spring table");
    }
    if (!rc) rc = cuda_check(cudaStreamSynchronize(ctx->stream), "cudaStreamSynchronize");
    if (rc) return rc;
    ctx->n_ranges += (long)rg.size();
    if (extend) {
        ctx->groups.back().n_meshes += n_meshes;
    } else {
        SpringGroup grp;
        grp.node_first = (int)ctx->n_nodes; grp.n_meshes = n_meshes; grp.nn = n_nodes;
        grp.off_first = (int)ctx->n_csr_off; grp.k = k;
        ctx->groups.push_back(grp);
        SpringGroupHost src;
        src.nn = n_nodes; src.k = k; src.rest = rest; src.edges.assign(h_edges, h_edges + (size_t)2 * n_edges);
        ctx->group_src.push_back(src);
        ctx->n_csr_off += (long)off.size();
        ctx->n_csr_ent += (long)ent.size();
    }
    ctx->h_orig.insert(ctx->h_orig.end(), og.begin(), og.end());
    ctx->h_stored.resize(ctx->h_orig.size());
    for (long m = ctx->n_nodes; m < ctx->n_nodes + add_nodes; ++m) ctx->h_stored[ctx->h_orig[m]] = (int)m;
    if (out_first_mesh_id) *out_first_mesh_id = (int)ctx->mesh_node_off.size() - 1;
    for (int s = 0; s < n_meshes; ++s) {
        ctx->n_nodes += n_nodes;
        ctx->n_edges += n_edges;
        ctx->mesh_node_off.push_back(ctx->n_nodes);
        ctx->mesh_edge_off.push_back(ctx->n_edges);
        ctx->mesh_constrained.push_back(0);
    }
    ctx->forces_valid = false;
    ctx->spread_current = false;
    return PLB_OK;
}

int ib_add_mesh(plb_ctx* ctx, int n_nodes, const double* h_xyz, int n_edges, const int* h_edges, const float* h_rest,
                float k, int* out_mesh_id) {
    return ib_add_meshes(ctx, 1, n_nodes, h_xyz, n_edges, h_edges, h_rest, k, out_mesh_id);
}

int ib_set_triangles(plb_ctx* ctx, int first_mesh_id, int n_meshes, int n_tris, const int* h_tris,
                     const double* h_ref_xyz, float k_s, float k_t, float k_v) {
    REQUIRE_CTX(ctx);
    const int total = (int)ctx->mesh_node_off.size() - 1;
    if (first_mesh_id < 0 || n_meshes < 1 || first_mesh_id + n_meshes > total || n_tris < 1 || !h_tris ||
        k_s < 0.f || k_t < 0.f || k_v < 0.f) {
        set_error("ib_set_triangles: invalid argument");
        return PLB_ERR_ARG;
    }
    const long nn = ctx->mesh_node_off[first_mesh_id + 1] - ctx->mesh_node_off[first_mesh_id];
    for (int s = 0; s < n_meshes; ++s) {
        if (ctx->mesh_node_off[first_mesh_id + s + 1] - ctx->mesh_node_off[first_mesh_id + s] != nn) {
            set_error("ib_set_triangles: meshes %d..%d do not share one topology", first_mesh_id, first_mesh_id + n_meshes - 1);
            return PLB_ERR_ARG;
        }
        if (ctx->mesh_constrained[first_mesh_id + s]) {
            set_error("ib_set_triangles: mesh %d already has triangles", first_mesh_id + s);
            return PLB_ERR_ORDER;
        }
    }
    for (int t = 0; t < 3 * n_tris; ++t)
        if (h_tris[t] < 0 || h_tris[t] >= nn) {
            set_error("ib_set_triangles: triangle %d has a node index out of range", t / 3);
            return PLB_ERR_ARG;
        }
    if (ctx->n_tris + (long)n_meshes * n_tris > ctx->cap_tris || ctx->n_cons + n_meshes > ctx->cap_cons) {
        set_error("ib_set_triangles: capacity exceeded (%ld/%ld triangles)", ctx->n_tris + (long)n_meshes * n_tris, ctx->cap_tris);
        return PLB_ERR_WORKSPACE;
    }
    // the unstressed shape: shared h_ref_xyz, or each mesh's current positions
    std::vector<double> cur;
    if (!h_ref_xyz) {
        cur.resize((size_t)3 * ctx->n_nodes);
        const int rc = ib_read_nodes(ctx, cur.data());
        if (rc && rc != PLB_ERR_NODE_LEFT) return rc;
    }
    std::vector<int4> tg((size_t)n_meshes * n_tris);
    std::vector<float> s0((size_t)n_meshes * n_tris);
    std::vector<MeshConstraint> mc((size_t)n_meshes);
    for (int s = 0; s < n_meshes; ++s) {
        const long noff = ctx->mesh_node_off[first_mesh_id + s];
        const double* ref = h_ref_xyz ? h_ref_xyz : cur.data() + 3 * noff;
        MeshConstraint& m = mc[s];
        reference_area_volume(ref, n_tris, h_tris, s0.data() + (size_t)s * n_tris, &m.S0_tot, &m.V0);
        for (int t = 0; t < n_tris; ++t) {
            if (!(s0[(size_t)s * n_tris + t] > 0.f)) {
                set_error("ib_set_triangles: triangle %d of the unstressed shape has zero area", t);
                return PLB_ERR_ARG;
            }
            tg[(size_t)s * n_tris + t] = make_int4(ctx->h_stored[noff + h_tris[3 * t]], ctx->h_stored[noff + h_tris[3 * t + 1]],
                                                   ctx->h_stored[noff + h_tris[3 * t + 2]], 0);
        }
        if (!(m.V0 > 0.0)) {
            set_error("ib_set_triangles: the surface is not closed or not oriented outwards (V_0 = %g)", m.V0);
            return PLB_ERR_ARG;
        }
        m.tri_first = (int)(ctx->n_tris + (long)s * n_tris);
        m.tri_count = n_tris;
        m.node_first = (int)noff;
        m.pad = 0; m.pad2 = 0.f;
        m.k_s = k_s; m.k_t = k_t; m.k_v = k_v;
    }
    int rc = cuda_check(cudaMemcpyAsync(ctx->tris + ctx->n_tris, tg.data(), tg.size() * sizeof(int4), cudaMemcpyHostToDevice, ctx->stream), "upload triangles");
    if (!rc) rc = cuda_check(cudaMemcpyAsync(ctx->tri_S0 + ctx->n_tris, s0.data(), s0.size() * sizeof(float), cudaMemcpyHostToDevice, ctx->stream), "upload triangle areas");
    if (!rc) rc = cuda_check(cudaMemcpyAsync(ctx->cons + ctx->n_cons, mc.data(), mc.size() * sizeof(MeshConstraint), cudaMemcpyHostToDevice, ctx->stream), "upload mesh constraints");
    if (!rc) rc = cuda_check(cudaStreamSynchronize(ctx->stream), "cudaStreamSynchronize");
    if (rc) return rc;
    ctx->n_tris += (long)n_meshes * n_tris;
    ctx->n_cons += n_meshes;
    for (int s = 0; s < n_meshes; ++s) ctx->mesh_constrained[first_mesh_id + s] = 1;
    ctx->forces_valid = false;
    return PLB_OK;
}

int ib_compute_membrane_forces(plb_ctx* ctx, float noise_sigma, unsigned long long noise_seed, unsigned long long step) {
    REQUIRE_CTX(ctx);
    if (noise_sigma < 0.f) {
        set_error("noise_sigma must be >= 0");
        return PLB_ERR_ARG;
    }
    ctx->forces_valid = true;
    return launch_membrane_forces(ctx, noise_sigma, noise_seed, step);
}

int ib_spread(plb_ctx* ctx, float* d_forcing) {
    REQUIRE_CTX(ctx);
    if (!d_forcing || ((uintptr_t)d_forcing & 15) != 0) {
        set_error("ib_spread: forcing buffer must be non-null and 16-byte aligned");
        return PLB_ERR_ARG;
    }
    if (ctx->n_nodes && !ctx->forces_valid) {
        set_error("ib_spread before ib_compute_membrane_forces");
        return PLB_ERR_ORDER;
    }
    // clear what the previous spread wrote (into whichever buffer it used) and drop its segment list
    const bool cleared = ctx->spread_target != nullptr;
    if (cleared) {
        const int rc = launch_clear_spread(ctx, ctx->spread_target);
        if (rc) return rc;
    }
    ctx->spread_target = (float4*)d_forcing;
    ctx->spread_current = true;
    // the spread kernel overlaps the clear up to its flush (programmatic dependent launch, ib.cu)
    return launch_spread(ctx, (float4*)d_forcing, cleared);
}

int ib_release_forcing(plb_ctx* ctx) {
    REQUIRE_CTX(ctx);
    int rc = PLB_OK;
    if (ctx->spread_target) rc = launch_clear_spread(ctx, ctx->spread_target);
    if (!rc) rc = cuda_check(cudaStreamSynchronize(ctx->stream), "cudaStreamSynchronize");
    ctx->spread_target = nullptr;
    ctx->spread_current = false;
    ctx->g_last = nullptr;
    ctx->g_last_mode = FORCE_NONE;
    return rc;
}

int ib_set_spread_mode(plb_ctx* ctx, int mode) {
    REQUIRE_CTX(ctx);
    if (mode != PLB_SPREAD_AUTO && mode != PLB_SPREAD_SCATTER && mode != PLB_SPREAD_AGGREGATE && mode != PLB_SPREAD_GATHER) {
        set_error("ib_set_spread_mode: unknown mode %d", mode);
        return PLB_ERR_ARG;
    }
    ctx->spread_mode = mode;
    return PLB_OK;
}

int ib_get_spread_mode(plb_ctx* ctx, int* out_mode_in_use) {
    REQUIRE_CTX(ctx);
    if (!out_mode_in_use) return PLB_ERR_ARG;
    *out_mode_in_use = spread_mode_of(ctx);
    return PLB_OK;
}

int ib_interpolate_advance(plb_ctx* ctx) {
    REQUIRE_CTX(ctx);
    if (ctx->n_nodes == 0) return PLB_OK;
    // no ib_spread needs to have run: lbm_step(NULL) -> ib_interpolate_advance is passive advection
    // (Eq. 33 alone); the force term of v is that of the last lbm_step, whatever its source
    if (!ctx->populated) {
        set_error("ib_interpolate_advance before the populations were set");
        return PLB_ERR_ORDER;
    }
    const int rc = launch_interpolate_advance(ctx);
    ctx->spread_current = false;
    ctx->forces_valid = false;
    return rc;
}

// ------------------------------------------------------------------------------------------------
// NEXT-4: adhesion.  The receptors, bonds and per-site tables live in their own caller-owned workspace.
static size_t carve_adhesion(Ctx* c, char* base, long n_sites, long n_rec) {
    Carve w{base, 0};
    int* rec_node = w.take<int>((size_t)n_rec);
    int4* bond = w.take<int4>((size_t)n_rec);
    int* site_count = w.take<int>((size_t)n_sites);
    int* site_min = w.take<int>((size_t)n_sites);
    if (c) {
        c->rec_node = rec_node; c->bond = bond; c->site_count = site_count; c->site_min = site_min;
    }
    return w.off;
}

static void tangential_axes(int a, int* t0, int* t1) {
    *t0 = a == 0 ? 1 : 0;
    *t1 = a == 2 ? 1 : 2;
}

int ib_adhesion_workspace_bytes(const plb_grid* grid, int wall_axis, long n_receptors, size_t* out_bytes) {
    long cells;
    int rc = check_grid(grid, &cells);
    if (rc) return rc;
    if (!out_bytes || wall_axis < 0 || wall_axis > 2 || n_receptors < 0) {
        set_error("ib_adhesion_workspace_bytes: invalid argument");
        return PLB_ERR_ARG;
    }
    const int n[3] = {grid->nx, grid->ny, grid->nz};
    int t0, t1;
    tangential_axes(wall_axis, &t0, &t1);
    *out_bytes = carve_adhesion(nullptr, nullptr, (long)n[t0] * n[t1], n_receptors);
    return PLB_OK;
}

int ib_set_receptors(plb_ctx* ctx, long n_receptors, const int* h_node, const plb_adhesion* prm, void* d_workspace,
                     size_t workspace_bytes) {
    REQUIRE_CTX(ctx);
    if (n_receptors < 0 || (n_receptors > 0 && !h_node) || !prm || !d_workspace || ((uintptr_t)d_workspace & 255) != 0) {
        set_error("ib_set_receptors: invalid argument (the workspace must be non-null and 256-byte aligned)");
        return PLB_ERR_ARG;
    }
    const int a = prm->wall_axis;
    if (a < 0 || a > 2 || ctx->bnd.kind[a] == PLB_PERIODIC) {
        set_error("ib_set_receptors: wall_axis %d is not a wall axis of this context", a);
        return PLB_ERR_ARG;
    }
    if (prm->max_per_site < 1 || prm->max_per_site > ADH_MAX_PER_SITE || !(prm->l_max > 0.f) || prm->k_on0 < 0.f ||
        prm->k_off0 < 0.f || prm->F0 < 0.f || prm->tau_rep < 0.f || (prm->F0 > 0.f && !(prm->tau_rep > 0.f))) {
        set_error("ib_set_receptors: invalid parameters (1 <= max_per_site <= %d, l_max > 0, rates, F0, tau_rep >= 0, tau_rep > 0 when F0 > 0)", ADH_MAX_PER_SITE);
        return PLB_ERR_ARG;
    }
    if (n_receptors >= (long)ADH_NO_OFFER) {
        set_error("ib_set_receptors: more than 0x7f7f7f7f receptors");
        return PLB_ERR_ARG;
    }
    for (long r = 0; r < n_receptors; ++r)
        if (h_node[r] < 0 || h_node[r] >= ctx->n_nodes) {
            set_error("ib_set_receptors: receptor %ld sits on node %d, out of range", r, h_node[r]);
            return PLB_ERR_ARG;
        }
    const int n[3] = {ctx->grid.nx, ctx->grid.ny, ctx->grid.nz};
    int t0, t1;
    tangential_axes(a, &t0, &t1);
    const long n_sites = (long)n[t0] * n[t1];
    const size_t need = carve_adhesion(nullptr, nullptr, n_sites, n_receptors);
    if (workspace_bytes < need) {
        set_error("ib_set_receptors: workspace of %zu bytes is smaller than the %zu needed", workspace_bytes, need);
        return PLB_ERR_WORKSPACE;
    }
    carve_adhesion(ctx, (char*)d_workspace, n_sites, n_receptors);
    AdhParams& p = ctx->adh;
    p.a = a; p.t0 = t0; p.t1 = t1; p.n0 = n[t0]; p.n1 = n[t1];
    p.per0 = ctx->bnd.kind[t0] == PLB_PERIODIC; p.per1 = ctx->bnd.kind[t1] == PLB_PERIODIC;
    p.max_per_site = prm->max_per_site;
    p.plane = ctx->bnd.kind[a] == PLB_WALL_HH ? 0.0 : -0.5;
    p.k_on0 = prm->k_on0; p.k_off0 = prm->k_off0; p.s = prm->s; p.gamma = prm->gamma; p.sigma = prm->sigma;
    p.l_b = prm->l_b; p.l_max = prm->l_max; p.F0 = prm->F0; p.tau_rep = prm->tau_rep;
    ctx->n_rec = n_receptors;
    ctx->adh_on = true;
    int rc = cuda_check(cudaMemsetAsync(d_workspace, 0, need, ctx->stream), "clear adhesion workspace");
    if (!rc) rc = cuda_check(cudaMemsetAsync(ctx->site_min, 0x7f, (size_t)n_sites * sizeof(int), ctx->stream), "reset site minima");
    std::vector<int> stored((size_t)n_receptors);
    for (long r = 0; r < n_receptors; ++r) stored[r] = ctx->h_stored[h_node[r]];
    if (!rc && n_receptors)
        rc = cuda_check(cudaMemcpyAsync(ctx->rec_node, stored.data(), (size_t)n_receptors * sizeof(int), cudaMemcpyHostToDevice,
                                        ctx->stream), "upload receptor nodes");
    if (!rc) rc = cuda_check(cudaStreamSynchronize(ctx->stream), "cudaStreamSynchronize");
    ctx->forces_valid = false;
    return rc;
}

int ib_adhesion_update(plb_ctx* ctx, unsigned long long seed, unsigned long long step) {
    REQUIRE_CTX(ctx);
    if (!ctx->adh_on) {
        set_error("ib_adhesion_update before ib_set_receptors");
        return PLB_ERR_ORDER;
    }
    ctx->forces_valid = false;
    return launch_adhesion_update(ctx, seed, step);
}

int ib_n_receptors(plb_ctx* ctx, long* out) {
    REQUIRE_CTX(ctx);
    if (!out) return PLB_ERR_ARG;
    *out = ctx->adh_on ? ctx->n_rec : 0;
    return PLB_OK;
}

int ib_read_bonds(plb_ctx* ctx, int* h_bonds) {
    REQUIRE_CTX(ctx);
    if (!h_bonds || !ctx->adh_on) {
        set_error("ib_read_bonds: null output or no receptors set");
        return h_bonds ? PLB_ERR_ORDER : PLB_ERR_ARG;
    }
    const long n = ctx->n_rec;
    std::vector<int4> tmp((size_t)n);
    int rc = PLB_OK;
    if (n) rc = cuda_check(cudaMemcpyAsync(tmp.data(), ctx->bond, (size_t)n * sizeof(int4), cudaMemcpyDeviceToHost, ctx->stream),
                           "download bonds");
    if (!rc) rc = sync_status(ctx);
    for (long r = 0; r < n; ++r) {
        h_bonds[3 * r] = tmp[r].x; h_bonds[3 * r + 1] = tmp[r].y; h_bonds[3 * r + 2] = tmp[r].z;
    }
    return rc;
}

int ib_write_bonds(plb_ctx* ctx, const int* h_bonds) {
    REQUIRE_CTX(ctx);
    if (!h_bonds || !ctx->adh_on) {
        set_error("ib_write_bonds: null input or no receptors set");
        return h_bonds ? PLB_ERR_ORDER : PLB_ERR_ARG;
    }
    const long n = ctx->n_rec;
    std::vector<int4> tmp((size_t)n);
    for (long r = 0; r < n; ++r) {
        const int on = h_bonds[3 * r] ? 1 : 0;
        tmp[r] = make_int4(on, on ? h_bonds[3 * r + 1] : 0, on ? h_bonds[3 * r + 2] : 0, -1);
        // a bond to a site outside a non-periodic tangential axis is refused here, before anything is
        // uploaded: left in the table, the next update would index the site counts out of bounds
        if (on && ((!ctx->adh.per0 && (tmp[r].y < 0 || tmp[r].y >= ctx->adh.n0)) ||
                   (!ctx->adh.per1 && (tmp[r].z < 0 || tmp[r].z >= ctx->adh.n1)))) {
            set_error("ib_write_bonds: receptor %ld is bound to site (%d, %d), outside a non-periodic tangential axis", r,
                      tmp[r].y, tmp[r].z);
            return PLB_ERR_ARG;
        }
    }
    int rc = PLB_OK;
    if (n) rc = cuda_check(cudaMemcpyAsync(ctx->bond, tmp.data(), (size_t)n * sizeof(int4), cudaMemcpyHostToDevice, ctx->stream),
                           "upload bonds");
    if (!rc) rc = launch_adhesion_recount(ctx);
    if (!rc) rc = sync_status(ctx);
    ctx->forces_valid = false;
    return rc;
}

// ------------------------------------------------------------------------------------------------
int ib_n_nodes(plb_ctx* ctx, long* out) {
    REQUIRE_CTX(ctx);
    if (!out) return PLB_ERR_ARG;
    *out = ctx->n_nodes;
    return PLB_OK;
}

int ib_read_nodes(plb_ctx* ctx, double* h_xyz) {
    REQUIRE_CTX(ctx);
    if (!h_xyz) return PLB_ERR_ARG;
    const long n = ctx->n_nodes;
    if (n) {
        // SoA -> AoS on the device, then one copy straight into the caller's buffer
        int rc = launch_nodes_transpose(ctx, /*to_aos=*/true);
        if (rc) return rc;
        rc = cuda_check(cudaMemcpyAsync(h_xyz, ctx->stage, (size_t)3 * n * sizeof(double), cudaMemcpyDeviceToHost,
                                        ctx->stream), "download node positions");
        if (rc) return rc;
    }
    return sync_status(ctx);
}

int ib_write_nodes(plb_ctx* ctx, const double* h_xyz) {
    REQUIRE_CTX(ctx);
    if (!h_xyz) return PLB_ERR_ARG;
    const long n = ctx->n_nodes;
    int rc = PLB_OK;
    if (n) {
        rc = cuda_check(cudaMemcpyAsync(ctx->stage, h_xyz, (size_t)3 * n * sizeof(double), cudaMemcpyHostToDevice,
                                        ctx->stream), "upload node positions");
        if (!rc) rc = launch_nodes_transpose(ctx, /*to_aos=*/false);
    }
    if (!rc) rc = cuda_check(cudaStreamSynchronize(ctx->stream), "cudaStreamSynchronize");
    ctx->forces_valid = false;
    ctx->spread_current = false;
    return rc;
}

static int read_node_float4(plb_ctx* ctx, const float4* d_src, float* h_out) {
    const long n = ctx->n_nodes;
    std::vector<float4> tmp((size_t)n);
    int rc = cuda_check(cudaMemcpyAsync(tmp.data(), d_src, (size_t)n * sizeof(float4), cudaMemcpyDeviceToHost, ctx->stream),
                        "download node data");
    if (!rc) rc = cuda_check(cudaStreamSynchronize(ctx->stream), "cudaStreamSynchronize");
    if (rc) return rc;
    for (long m = 0; m < n; ++m) {
        const long o = ctx->h_orig[m];
        h_out[3 * o] = tmp[m].x; h_out[3 * o + 1] = tmp[m].y; h_out[3 * o + 2] = tmp[m].z;
    }
    return PLB_OK;
}

int ib_read_forces(plb_ctx* ctx, float* h_F) {
    REQUIRE_CTX(ctx);
    if (!h_F) return PLB_ERR_ARG;
    return read_node_float4(ctx, ctx->F, h_F);
}

int ib_read_node_velocities(plb_ctx* ctx, float* h_U) {
    REQUIRE_CTX(ctx);
    if (!h_U) return PLB_ERR_ARG;
    return read_node_float4(ctx, ctx->U, h_U);
}

int ib_write_forces(plb_ctx* ctx, const float* h_F) {
    REQUIRE_CTX(ctx);
    if (!h_F) return PLB_ERR_ARG;
    const long n = ctx->n_nodes;
    std::vector<float4> tmp((size_t)n);
    for (long m = 0; m < n; ++m) {
        const long o = ctx->h_orig[m];
        tmp[m] = make_float4(h_F[3 * o], h_F[3 * o + 1], h_F[3 * o + 2], 0.f);
    }
    int rc = cuda_check(cudaMemcpyAsync(ctx->F, tmp.data(), (size_t)n * sizeof(float4), cudaMemcpyHostToDevice, ctx->stream),
                        "upload forces");
    if (!rc) rc = cuda_check(cudaStreamSynchronize(ctx->stream), "cudaStreamSynchronize");
    ctx->forces_valid = true;
    return rc;
}

int lbm_check_finite(plb_ctx* ctx, long* out_bad_cells) {
    REQUIRE_CTX(ctx);
    if (!out_bad_cells || !ctx->populated) {
        set_error("lbm_check_finite: null output or populations not set");
        return out_bad_cells ? PLB_ERR_ORDER : PLB_ERR_ARG;
    }
    int* d_bad = ctx->counters + 8;                    // scratch counter
    int rc = cuda_check(cudaMemsetAsync(d_bad, 0, sizeof(int), ctx->stream), "clear counter");
    if (!rc) rc = launch_check_finite(ctx, d_bad);
    int h = 0;
    if (!rc) rc = cuda_check(cudaMemcpyAsync(&h, d_bad, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream), "read counter");
    if (!rc) rc = cuda_check(cudaStreamSynchronize(ctx->stream), "cudaStreamSynchronize");
    *out_bad_cells = h;
    return rc;
}

int lbm_check_finite_static(plb_ctx* ctx, int* d_out_bad_cells) {
    REQUIRE_CTX(ctx);
    if (!d_out_bad_cells || !ctx->populated) {
        set_error("lbm_check_finite_static: null output or populations not set");
        return d_out_bad_cells ? PLB_ERR_ORDER : PLB_ERR_ARG;
    }
    return launch_check_finite_static(ctx, d_out_bad_cells);
}

int plb_status(plb_ctx* ctx) {
    REQUIRE_CTX(ctx);
    return sync_status(ctx);
}

int plb_launch_count(plb_ctx* ctx, long* out) {
    REQUIRE_CTX(ctx);
    if (!out) return PLB_ERR_ARG;
    *out = ctx->launches;
    return PLB_OK;
}

int plb_philox4x32_10(void* cuda_stream, long n, const unsigned* d_ctr, const unsigned* d_key, unsigned* d_out) {
    if (n < 0 || (n > 0 && (!d_ctr || !d_key || !d_out))) {
        set_error("plb_philox4x32_10: invalid argument");
        return PLB_ERR_ARG;
    }
    return launch_philox((cudaStream_t)cuda_stream, n, d_ctr, d_key, d_out);
}

}  // extern "C"
