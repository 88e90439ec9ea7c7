// adhesion.cu -- SURVEY.md NEXT-4: the stochastic dynamic adhesion model (section 3.2,
// Eq. 12-14, rules L147-149, P_f / P_r L151) and the short-range wall repulsion (section 3.4.1,
// L244-246), the step after S5 in the paper's loop (L276).  The paper's own kernel
// (sem_platelet_wall_kernel, L364-373) is "one thread per receptor"; so is this one, with the
// contention for the places of a vWF site resolved deterministically (lowest receptor index first)
// instead of by arrival order, for any number of same-step candidates per site.
//
// Monte-Carlo decisions are integer outcomes: the probabilities and the capture test are evaluated
// in fp64 (B200 has full-rate-enough fp64 for a few million receptors), the same precision the
// reference computation uses, so that both take the same decision from the same uniform.
#include "plb_internal.cuh"

namespace plb {

__device__ __forceinline__ long adh_site_index(const AdhParams& p, long s0, long s1) {
    if (p.per0) { s0 %= p.n0; if (s0 < 0) s0 += p.n0; } else if (s0 < 0 || s0 >= p.n0) return -1;
    if (p.per1) { s1 %= p.n1; if (s1 < 0) s1 += p.n1; } else if (s1 < 0 || s1 >= p.n1) return -1;
    return s0 + (long)p.n0 * s1;
}

struct NodePos { double w, t0, t1; };   // wall-normal and the two tangential coordinates

__device__ __forceinline__ NodePos adh_node(const AdhParams& p, const double* const* X, const int m) {
    NodePos q;
    q.w = X[p.a][m]; q.t0 = X[p.t0][m]; q.t1 = X[p.t1][m];
    return q;
}

struct NodeArrays { const double* X[3]; };

// d = |x_b - l_b|;  k_on = k_on0 exp(s d (gamma - d/2)) (Eq. 13);  k_off = k_off0 exp(gamma s d) (Eq. 12)
__device__ __forceinline__ double adh_P_form(const AdhParams& p, const double x_b) {
    const double d = fabs(x_b - p.l_b);
    return 1.0 - exp(-(p.k_on0 * exp(p.s * d * (p.gamma - 0.5 * d))));
}
__device__ __forceinline__ double adh_P_break(const AdhParams& p, const double x_b) {
    const double d = fabs(x_b - p.l_b);
    return 1.0 - exp(-(p.k_off0 * exp(p.gamma * p.s * d)));
}
__device__ __forceinline__ double adh_uniform(const uint32_t r) {      // ((r >> 8) + 1/2) 2^-24
    return ((double)(r >> 8) + 0.5) * (1.0 / 16777216.0);
}

// pass 1, one thread per receptor: break test of an existing bond, then (if the receptor is or has
// just become unbound) formation test against its nearest site; a receptor that passes the
// formation test becomes a candidate of the site.  bond = (bound, s0, s1, candidate site or -1)
__global__ void __launch_bounds__(256) adhesion_test_kernel(const NodeArrays nodes, const int* __restrict__ rec_node,
                                                            int4* __restrict__ bond, int* __restrict__ site_count,
                                                            const long n_rec, const AdhParams p,
                                                            const unsigned long long seed, const unsigned step) {
    const long r = blockIdx.x * 256L + threadIdx.x;
    if (r >= n_rec) return;
    int4 b = bond[r];
    const NodePos q = adh_node(p, nodes.X, __ldg(rec_node + r));
    const uint4 w = noise_words(seed, (unsigned long long)r, step, 3u);
    const double hw = p.plane - q.w;
    if (b.x) {
        const double r0 = (double)b.y - q.t0, r1 = (double)b.z - q.t1;
        const double x_b = sqrt(hw * hw + r0 * r0 + r1 * r1);
        if (adh_uniform(w.x) < adh_P_break(p, x_b)) {
            b.x = 0;
            atomicSub(site_count + adh_site_index(p, b.y, b.z), 1);
        }
    }
    b.w = -1;
    if (!b.x) {
        b.y = 0; b.z = 0;
        const long s0 = (long)floor(q.t0 + 0.5), s1 = (long)floor(q.t1 + 0.5);      // nearest site
        const long si = adh_site_index(p, s0, s1);
        if (si >= 0) {
            const double r0 = (double)s0 - q.t0, r1 = (double)s1 - q.t1;
            const double x_b = sqrt(hw * hw + r0 * r0 + r1 * r1);
            if (x_b < p.l_max && adh_uniform(w.y) < adh_P_form(p, x_b)) {
                b.y = (int)s0; b.z = (int)s1; b.w = (int)si;
            }
        }
    }
    bond[r] = b;
}

// passes 2 .. : the places of a site go to its candidates in the order of their receptor index (rule
// 2 of L148 read as a sweep in index order, A-7), however many candidates there are.
// One ROUND gives every site with candidates one decision: every pending candidate offers its
// index to its site by atomicMin, then the candidate that sees its own index has the lowest one
// left; it binds if the site still has a free place, and leaves the contest either way.  A site
// can take at most max_per_site bonds, so after max_per_site rounds every candidate still pending
// belongs to a full site and loses (last = true).
__global__ void __launch_bounds__(256) adhesion_offer_kernel(const int4* __restrict__ bond, int* __restrict__ site_min,
                                                             const long n_rec) {
    const long r = blockIdx.x * 256L + threadIdx.x;
    if (r >= n_rec) return;
    const int si = bond[r].w;
    if (si >= 0) atomicMin(site_min + si, (int)r);
}

__global__ void __launch_bounds__(256) adhesion_award_kernel(int4* __restrict__ bond, int* __restrict__ site_count,
                                                             int* __restrict__ site_min, const long n_rec,
                                                             const int max_per_site, const bool last) {
    const long r = blockIdx.x * 256L + threadIdx.x;
    if (r >= n_rec) return;
    int4 b = bond[r];
    if (b.w < 0) return;
    if (site_min[b.w] == (int)r) {                       // the only thread that touches this site now
        const int held = site_count[b.w];
        if (held < max_per_site) { b.x = 1; site_count[b.w] = held + 1; }
        else { b.y = 0; b.z = 0; }
        b.w = -1;
    } else if (last) {
        b.y = 0; b.z = 0; b.w = -1;
    }
    bond[r] = b;
}

// between two rounds: the minimum of a site that just decided is forgotten (its winner no longer
// offers); one thread per receptor that decided would race with the readers above, so this is a
// pass of its own over the candidates still pending
__global__ void __launch_bounds__(256) adhesion_reset_kernel(const int4* __restrict__ bond, int* __restrict__ site_min,
                                                             const long n_rec) {
    const long r = blockIdx.x * 256L + threadIdx.x;
    if (r >= n_rec) return;
    const int si = bond[r].w;
    if (si >= 0) site_min[si] = ADH_NO_OFFER;
}

// per-site bond counts from the bond table (ib_write_bonds)
__global__ void __launch_bounds__(256) adhesion_count_kernel(const int4* __restrict__ bond, int* __restrict__ site_count,
                                                             int* __restrict__ counters, const long n_rec, const AdhParams p) {
    const long r = blockIdx.x * 256L + threadIdx.x;
    if (r >= n_rec) return;
    const int4 b = bond[r];
    if (!b.x) return;
    const long si = adh_site_index(p, b.y, b.z);
    if (si < 0) atomicOr(counters + 1, STATUS_ADH_BAD_SITE);
    else atomicAdd(site_count + si, 1);
}

// Eq. 14: the bond pulls its node towards the site with sigma (x_b - l_b) (pushes when compressed)
__global__ void __launch_bounds__(256) adhesion_force_kernel(const NodeArrays nodes, const int* __restrict__ rec_node,
                                                             const int4* __restrict__ bond, float4* __restrict__ F,
                                                             const long n_rec, const AdhParams p) {
    const long r = blockIdx.x * 256L + threadIdx.x;
    if (r >= n_rec) return;
    const int4 b = bond[r];
    if (!b.x) return;
    const int m = __ldg(rec_node + r);
    const NodePos q = adh_node(p, nodes.X, m);
    double R[3];
    R[p.a] = p.plane - q.w; R[p.t0] = (double)b.y - q.t0; R[p.t1] = (double)b.z - q.t1;
    const double x_b = sqrt(R[0] * R[0] + R[1] * R[1] + R[2] * R[2]);
    if (!(x_b > 0.0)) return;
    const double f = p.sigma * (x_b - p.l_b) / x_b;
    atomicAdd(F + m, make_float4((float)(f * R[0]), (float)(f * R[1]), (float)(f * R[2]), 0.f));
}

// L246: F_rep = F0 tau exp(-tau eps)/(1 - exp(-tau eps)) on every node, along the inward normal
__global__ void __launch_bounds__(256) wall_repulsion_kernel(const double* __restrict__ Xw, float4* __restrict__ F,
                                                             int* __restrict__ counters, const long n_nodes, const AdhParams p) {
    const long m = blockIdx.x * 256L + threadIdx.x;
    if (m >= n_nodes) return;
    const double eps = Xw[m] - p.plane;
    if (!(eps > 0.0)) {
        atomicOr(counters + 1, STATUS_NODE_LEFT);
        return;
    }
    const double e = exp(-p.tau_rep * eps);
    const float fr = (float)(p.F0 * p.tau_rep * e / (1.0 - e));
    float4 f = F[m];
    if (p.a == 0) f.x += fr; else if (p.a == 1) f.y += fr; else f.z += fr;
    F[m] = f;
}

static NodeArrays node_arrays(const Ctx* c) {
    NodeArrays n;
    n.X[0] = c->X[0]; n.X[1] = c->X[1]; n.X[2] = c->X[2];
    return n;
}
static unsigned blocks_for(long n) { return (unsigned)((n + 255) / 256); }

int launch_adhesion_forces(Ctx* c) {
    if (!c->adh_on) return PLB_OK;
    if (c->n_rec) {
        adhesion_force_kernel<<<blocks_for(c->n_rec), 256, 0, c->stream>>>(node_arrays(c), c->rec_node, c->bond, c->F,
                                                                          c->n_rec, c->adh);
        c->launches++;
    }
    if (c->adh.F0 > 0.0 && c->n_nodes) {
        wall_repulsion_kernel<<<blocks_for(c->n_nodes), 256, 0, c->stream>>>(c->X[c->adh.a], c->F, c->counters, c->n_nodes,
                                                                            c->adh);
        c->launches++;
    }
    return cuda_check(cudaGetLastError(), "adhesion force kernels");
}

int launch_adhesion_update(Ctx* c, unsigned long long seed, unsigned long long step) {
    if (!c->n_rec) return PLB_OK;
    const unsigned grid = blocks_for(c->n_rec);
    adhesion_test_kernel<<<grid, 256, 0, c->stream>>>(node_arrays(c), c->rec_node, c->bond, c->site_count, c->n_rec, c->adh,
                                                      seed, (unsigned)step);
    c->launches++;
    // site_min is INT_MAX everywhere between updates (set at ib_set_receptors; every site that was
    // offered to is reset below or decided for good in the last round)
    const int rounds = c->adh.max_per_site;
    for (int round = 0; round < rounds; ++round) {
        adhesion_offer_kernel<<<grid, 256, 0, c->stream>>>(c->bond, c->site_min, c->n_rec);
        adhesion_award_kernel<<<grid, 256, 0, c->stream>>>(c->bond, c->site_count, c->site_min, c->n_rec,
                                                           c->adh.max_per_site, round == rounds - 1);
        c->launches += 2;
        if (round < rounds - 1) {
            adhesion_reset_kernel<<<grid, 256, 0, c->stream>>>(c->bond, c->site_min, c->n_rec);
            c->launches++;
        }
    }
    // the sites decided in the last round still hold their winner's index
    int rc = cuda_check(cudaMemsetAsync(c->site_min, 0x7f, (size_t)c->adh.n0 * c->adh.n1 * sizeof(int), c->stream),
                        "reset site minima");
    if (rc) return rc;
    return cuda_check(cudaGetLastError(), "adhesion update kernels");
}

int launch_adhesion_recount(Ctx* c) {
    int rc = cuda_check(cudaMemsetAsync(c->site_count, 0, (size_t)c->adh.n0 * c->adh.n1 * sizeof(int), c->stream),
                        "clear site counts");
    if (rc || !c->n_rec) return rc;
    adhesion_count_kernel<<<blocks_for(c->n_rec), 256, 0, c->stream>>>(c->bond, c->site_count, c->counters, c->n_rec, c->adh);
    c->launches++;
    return cuda_check(cudaGetLastError(), "adhesion_count_kernel");
}

}  // namespace plb
