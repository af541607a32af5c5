// vmg_cluster.cuh -- S5 widened by one level: the level above the single-CTA tail runs DISTRIBUTED over a thread-block
// cluster, resident in the CTAs' shared memory for the whole down-stroke and up-stroke, with its halo planes exchanged
// through distributed shared memory and barrier.cluster between colour half-sweeps instead of kernel launches
// (SURVEY.md 7 step 7 "single-CTA (or one thread-block cluster with DSMEM) kernel"; hard part 1: coarse-level latency).
//
// Level D (e.g. 32x16x16 of the 256x128x128 hierarchy: 13 launches of ~1.9 us each as graph nodes) is cut into z-slabs of P
// planes, one per CTA of the cluster (P even: a CTA owns whole coarse planes).  Each CTA keeps its slab in the same
// natural-layout shared-memory block a tail level uses (six arrays with zero guards); the guards of phi, which are at
// least one plane long, double as the HALO planes, and the plane of wz above the slab is loaded once.  A thread relaxes
// the same two cells (one per colour) in every sweep with their weights, 1/D and rhs in registers (tail_smooth's scheme);
// a cell of the slab's first / last plane is also stored into the neighbour CTA's halo (st.shared::cluster through
// cluster.map_shared_rank), then the cluster synchronises.  Residual + restriction writes the coarse right-hand side to
// global memory, rank 0 runs the levels below as coarse_tail_body does (the other CTAs wait at a cluster barrier), the
// correction comes back through global memory, and the post-smoothing runs distributed again.
// Same expressions, same order as the per-step kernels: bitwise the plain launches it replaces.
#pragma once
#include <cooperative_groups.h>
#include "vmg_tail.cuh"

namespace vmg {

namespace cg = cooperative_groups;

struct ClusterArgs {
    TailArgs tail;     // the levels below D (lev[0] = D's child), run by rank 0 exactly as coarse_tail_kernel runs them
    TailLevel D;       // the distributed level: global arrays, full dimensions; D.off = offset of its block in shared memory
    int P;             // planes per CTA (even); cluster size = D.nz / P
};

// nsweeps red-black sweeps on the slab of this CTA; s / L: the slab as a tail level (nz = P); lo / hi: the phi blocks of
// the CTAs that own the planes below / above (nullptr at the domain faces)
__device__ __forceinline__ void cluster_smooth(cg::cluster_group& cl, const TailSmem& s, const TailLevel& L, double* lo, double* hi,
                                               int nsweeps, int first)
{
    const int hx = (L.nx + 1) >> 1;
    const int nt = hx * L.ny * L.nz;           // <= blockDim.x (plan_schedule)
    const int t = threadIdx.x;
    int c[2] = {-1, -1};
    int kk = 0;
    if (t < nt) {
        const int m = t % hx, j = (t / hx) % L.ny;
        kk = t / (hx * L.ny);
#pragma unroll
        for (int colour = 0; colour < 2; ++colour) {
            const int i = 2 * m + ((colour + j + kk) & 1);      // the slab starts at an even plane: local parity = global parity
            if (i < L.nx) c[colour] = i + L.nx * j + L.nxy * kk;
        }
        if (first) { const int tmp = c[0]; c[0] = c[1]; c[1] = tmp; }
    }
    double w[2][6], di[2], rh[2];
    int cc[2];
#pragma unroll
    for (int q = 0; q < 2; ++q) {
        cc[q] = c[q] >= 0 ? c[q] : 0;
        w[q][0] = s.wx[cc[q]]; w[q][1] = s.wx[cc[q] + 1];
        w[q][2] = s.wy[cc[q]]; w[q][3] = s.wy[cc[q] + L.nx];
        w[q][4] = s.wz[cc[q]]; w[q][5] = s.wz[cc[q] + L.zs];
        di[q] = s.dinv[cc[q]]; rh[q] = s.rhs[cc[q]];
    }
    const int nx = L.nx, zs = L.zs, nloc = L.n;
    double* const ph = s.phi;
    // where a relaxed cell goes besides its own place: the upper halo of the CTA below (first plane of the slab), the lower
    // halo of the CTA above (last plane)
    double* push[2] = {nullptr, nullptr};
#pragma unroll
    for (int q = 0; q < 2; ++q) {
        if (c[q] < 0) continue;
        const int in_plane = c[q] - L.nxy * kk;
        if (kk == 0 && lo) push[q] = lo + nloc + in_plane;
        if (kk == L.nz - 1 && hi) push[q] = hi - L.nxy + in_plane;       // (P >= 2: a cell is never in both)
    }
    for (int sw = 0; sw < nsweeps; ++sw) {
#pragma unroll
        for (int q = 0; q < 2; ++q) {
            if (c[q] >= 0) {
                double* const x = ph + cc[q];
                const double a0 = x[-1], a1 = x[1], a2 = x[-nx], a3 = x[nx], a4 = x[-zs], a5 = x[zs];
                double v = w[q][0] * a0;
                v = fma(w[q][1], a1, v);
                v = fma(w[q][2], a2, v);
                v = fma(w[q][3], a3, v);
                v = fma(w[q][4], a4, v);
                v = fma(w[q][5], a5, v);
                v = di[q] * (rh[q] + v);
                *x = v;
                if (push[q]) *push[q] = v;
            }
            cl.sync();
        }
    }
}

template <int NT>
__global__ void __launch_bounds__(NT, 1) coarse_cluster_kernel(ClusterArgs g)
{
    grid_dependency_wait();
    extern __shared__ __align__(16) double tail_smem[];
    cg::cluster_group cl = cg::this_cluster();
    const int rank = (int)cl.block_rank(), nc = (int)cl.num_blocks();
    const int tid = threadIdx.x, nth = blockDim.x;
    const long long off = (long long)(blockIdx.x / nc) * g.tail.pstride;      // one cluster per problem of a batched launch

    // the slab as a tail level of P planes
    TailLevel L = g.D;
    L.nz = g.P; L.n = L.nxy * g.P;
    const TailLevel& C = g.tail.lev[0];
    TailSmem s(tail_smem, L);
    const int st = tail_stride(L.n, L.guard);
    const int k0 = rank * g.P;

    if (rank == 0) TAIL_MARK(41);
    // ---- stage in: zero the slab's block (guards, halos, phi = 0: level D starts every cycle from zero), load its arrays ----
    for (int t = tid; t < 6 * st; t += nth) tail_smem[L.off + t] = 0.0;
    __syncthreads();
    for (int t = tid; t < L.n; t += nth) {
        const int i = t % L.nx, j = (t / L.nx) % L.ny, kk = t / L.nxy;
        const long long c = off + cell_at(g.D.G, i, j, k0 + kk);
        s.dinv[t] = g.D.dinv[c]; s.wx[t] = g.D.wx[c]; s.wy[t] = g.D.wy[c]; s.wz[t] = g.D.wz[c]; s.rhs[t] = g.D.rhs[c];
    }
    if (k0 + g.P < g.D.nz)                                   // the low-z face weights of the plane above the slab
        for (int t = tid; t < L.nxy; t += nth)
            s.wz[L.n + t] = g.D.wz[off + cell_at(g.D.G, t % L.nx, t / L.nx, k0 + g.P)];
    double* lo = rank > 0 ? cl.map_shared_rank(s.phi, rank - 1) : nullptr;
    double* hi = rank + 1 < nc ? cl.map_shared_rank(s.phi, rank + 1) : nullptr;
    cl.sync();                                               // every CTA's block is initialised before anyone pushes into it

    if (rank == 0) TAIL_MARK(42);
    // ---- down-stroke of level D ----
    cluster_smooth(cl, s, L, lo, hi, g.tail.nu1, 0);
    if (rank == 0) TAIL_MARK(43);
    {
        // residual + restriction (same order as residual_restrict_kernel); the coarse level lives in global memory here
        const int cnxy = C.nx * C.ny, ncoarse = cnxy * (g.P / 2);
        for (int t = tid; t < ncoarse; t += nth) {
            const int I = t % C.nx, J = (t / C.nx) % C.ny, Kl = t / cnxy;
            double acc = 0.0;
            for (int r = 0; r < 2; ++r)
                for (int q = 0; q < 2; ++q) {
                    const int cc = (2 * I) + L.nx * (2 * J + q) + L.nxy * (2 * Kl + r);
                    acc += tail_residual_at(s, L, cc) + tail_residual_at(s, L, cc + 1);
                }
            const long long gc = off + cell_at(C.G, I, J, k0 / 2 + Kl);
            C.rhs[gc] = acc / 8.0;
            C.phi[gc] = 0.0;
        }
    }
    __threadfence();
    cl.sync();

    if (rank == 0) TAIL_MARK(44);
    // ---- the levels below, by rank 0 alone ----
    if (rank == 0) coarse_tail_body(g.tail, off);
    __threadfence();
    cl.sync();

    if (rank == 0) TAIL_MARK(45);
    // ---- up-stroke of level D: correction from the child level (global), halo refresh, post-smoothing ----
    for (int t = tid; t < L.n; t += nth) {
        const int i = t % L.nx, j = (t / L.nx) % L.ny, kk = t / L.nxy;
        const double v = s.phi[t] + C.phi[off + cell_at(C.G, i >> 1, j >> 1, (k0 + kk) >> 1)];
        s.phi[t] = v;
        if (kk == 0 && lo) lo[L.n + (t - L.nxy * kk)] = v;
        if (kk == L.nz - 1 && hi) hi[-L.nxy + (t - L.nxy * kk)] = v;
    }
    cl.sync();
    if (rank == 0) TAIL_MARK(46);
    cluster_smooth(cl, s, L, lo, hi, g.tail.nu2, g.tail.sym);
    if (rank == 0) TAIL_MARK(47);

    // ---- stage out ----
    for (int t = tid; t < L.n; t += nth)
        g.D.phi[off + cell_at(g.D.G, t % L.nx, (t / L.nx) % L.ny, k0 + t / L.nxy)] = s.phi[t];
    if (rank == 0) TAIL_MARK(48);
}

}  // namespace vmg
