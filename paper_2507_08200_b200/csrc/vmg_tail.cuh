// vmg_tail.cuh -- S5: the coarse tail of the V-cycle in ONE CTA (north_star (3): "a single-CTA smoother";
// SURVEY.md 8(a) S5).  Every level from `first` down to the bottom lives in shared memory for the whole
// launch: pre-smoothing, residual+restriction, the fixed-sweep bottom solve (R11), prolongation+correction and
// post-smoothing run back to back with __syncthreads() between colour half-sweeps instead of kernel launches.
// The arithmetic of every step is the same expression, in the same order, as the per-step kernels of
// vmg_kernels.cuh, so the tail is bitwise identical to the plain launches it replaces.
#pragma once
#include "vmg_kernels.cuh"

namespace vmg {

constexpr int kTailMaxLevels = 12;
constexpr int kTailThreads = 1024;

struct TailLevel {
    const double *wx, *wy, *wz, *dinv;   // global, internal stencil form (cell 0)
    double *phi, *rhs;                   // global level arrays (cell 0)
    int nx, ny, nz, n, nxy, guard, off;  // off: offset (doubles) of this level's block in shared memory
    Geom G;                              // layout of the global arrays (shared memory uses the natural layout)
    int zs;                              // stride to the z neighbours: nxy in 3-D, 0 in 2-D (their weight is zero)
};

struct TailArgs {
    TailLevel lev[kTailMaxLevels];
    int nl;                    // levels in the tail; lev[nl-1] is the bottom
    int nu1, nu2, nbottom, sz; // sz = 2 in 3-D, 1 in 2-D (children per coarse cell along z)
    int prolong;               // 0: piecewise constant, 1: trilinear (R9 option)
    int sym;                   // 1: symmetric V-cycle: post-smoothing and the second half of the bottom sweeps black->red
    ProlongBC bc;              // boundary types (trilinear ghosts)
    int whole;                 // 1: lev[0] is level 0 of the hierarchy (phi is an initial guess, not zero)
    unsigned long long* norm_out;   // whole == 1: ||rhs - A phi||_inf bits after the cycle (may be NULL)
    long long pstride;         // batched launch (one CTA per problem): the arrays of problem blockIdx.x lie blockIdx.x * pstride doubles on
    const double* S;           // the bottom solve as a matrix (bottom_matrix_kernel; NULL: run the sweeps), row-major lev[nl-1].n squared
};

constexpr int kBottomMatrixMax = 64;   // largest bottom grid (cells) whose solve is kept as a matrix

// R11 says "nbottom red-black sweeps from a zero field": a fixed linear map of the right-hand side.  Column `blockIdx.x` of
// its matrix = the sweeps run on the unit vector e_col, one thread per cell of the bottom grid (<= 64 cells), the field in
// shared memory.  Built once per coefficient change (ready() in vmg_api.cu); the tail then replaces 2 nbottom dependent
// half-sweeps (16 k clk of the single-CTA kernel for the 4 x 2 x 2 bottom of config 3) by n fused multiply-adds per cell.
// Same map, different rounding order than the sweeps (the oracle runs the sweeps): covered by the 1e-10 / 1e-6 bars.
__global__ void bottom_matrix_kernel(const double* __restrict__ wx, const double* __restrict__ wy, const double* __restrict__ wz,
                                     const double* __restrict__ dinv, Geom G, int three_d, int nbottom, double* __restrict__ S)
{
    __shared__ double phi[kBottomMatrixMax];
    const int n = (int)G.n, t = threadIdx.x, col = blockIdx.x;
    int i = 0, j = 0, k = 0;
    double w[6] = {0, 0, 0, 0, 0, 0}, di = 0.0;
    int nb[6] = {0, 0, 0, 0, 0, 0};
    if (t < n) {
        i = t % G.nx; j = (t / G.nx) % G.ny; k = t / (G.nx * G.ny);
        const long long c = cell_at(G, i, j, k);
        di = dinv[c];
        // a face on the domain boundary carries a zero weight in the internal arrays (vmg_internal.h); the high faces are the
        // low faces of the neighbours
        if (i > 0)        { w[0] = wx[c];                        nb[0] = t - 1; }
        if (i < G.nx - 1) { w[1] = wx[cell_at(G, i + 1, j, k)];  nb[1] = t + 1; }
        if (j > 0)        { w[2] = wy[c];                        nb[2] = t - G.nx; }
        if (j < G.ny - 1) { w[3] = wy[cell_at(G, i, j + 1, k)];  nb[3] = t + G.nx; }
        if (three_d) {
            if (k > 0)        { w[4] = wz[c];                       nb[4] = t - G.nx * G.ny; }
            if (k < G.nz - 1) { w[5] = wz[cell_at(G, i, j, k + 1)]; nb[5] = t + G.nx * G.ny; }
        }
        phi[t] = 0.0;
    }
    const double rhs = t == col ? 1.0 : 0.0;
    __syncthreads();
    for (int s = 0; s < nbottom; ++s)
        for (int colour = 0; colour < 2; ++colour) {
            if (t < n && ((i + j + k) & 1) == colour) {
                double v = w[0] * phi[nb[0]];
                v = fma(w[1], phi[nb[1]], v);
                v = fma(w[2], phi[nb[2]], v);
                v = fma(w[3], phi[nb[3]], v);
                v = fma(w[4], phi[nb[4]], v);
                v = fma(w[5], phi[nb[5]], v);
                phi[t] = di * (rhs + v);
            }
            __syncthreads();
        }
    if (t < n) S[(long long)t * n + col] = phi[t];
}

// shared-memory block of a level: six arrays (phi, rhs, dinv, wx, wy, wz), each `guard` zeroed doubles, n cells,
// `guard` zeroed doubles; guard >= zs + nx + 2 so that every stencil neighbour of every cell is addressable
// and every out-of-domain neighbour meets a zero weight (same convention as the global arrays).
__host__ __device__ inline int tail_stride(int n, int guard) { return ((n + 2 * guard + 3) / 4) * 4; }
__host__ __device__ inline int tail_level_doubles(int n, int guard) { return 6 * tail_stride(n, guard); }

struct TailSmem {
    double *phi, *rhs, *dinv, *wx, *wy, *wz;
    __device__ TailSmem(double* base, const TailLevel& L)
    {
        int st = tail_stride(L.n, L.guard);
        double* p = base + L.off + L.guard;
        phi = p; rhs = p + st; dinv = p + 2 * st; wx = p + 3 * st; wy = p + 4 * st; wz = p + 5 * st;
    }
};

// natural-layout index of a shared-memory level (trilinear_value's accessor)
__device__ inline long long at_tail(const void* l, int i, int j, int k)
{
    const TailLevel& L = *(const TailLevel*)l;
    return i + L.nx * (j + L.ny * k);
}

__device__ __forceinline__ double tail_nb_sum(const TailSmem& s, const TailLevel& L, int c)
{
    double v = s.wx[c] * s.phi[c - 1];
    v = fma(s.wx[c + 1], s.phi[c + 1], v);
    v = fma(s.wy[c], s.phi[c - L.nx], v);
    v = fma(s.wy[c + L.nx], s.phi[c + L.nx], v);
    v = fma(s.wz[c], s.phi[c - L.zs], v);
    v = fma(s.wz[c + L.zs], s.phi[c + L.zs], v);
    return v;
}

// nsweeps red-black sweeps.  Levels whose half-sweep fits the CTA (nt <= blockDim: all tail levels in practice) take
// their cell indices once, not per half-sweep; levels whose half-sweep fits ONE WARP (the 32-sweep bottom solve on
// 4x2x2 or 2x2x2: 8 or 4 relaxations per colour) are relaxed by warp 0 alone with __syncwarp() between the colours
// instead of 64 block-wide barriers.  The caller's __syncthreads() semantics are kept: all threads leave in step.
__device__ __forceinline__ void tail_smooth(const TailSmem& s, const TailLevel& L, int nsweeps, int first = 0)
{
    const int hx = (L.nx + 1) >> 1;
    const int nt = hx * L.ny * L.nz;
    if (nt <= (int)blockDim.x) {
        const int t = threadIdx.x;
        int c[2] = {-1, -1};
        if (t < nt) {
            const int m = t % hx, j = (t / hx) % L.ny, k = t / (hx * L.ny);
#pragma unroll
            for (int colour = 0; colour < 2; ++colour) {
                const int i = 2 * m + ((colour + j + k) & 1);
                if (i < L.nx) c[colour] = i + L.nx * j + L.nxy * k;
            }
            if (first) { const int tmp = c[0]; c[0] = c[1]; c[1] = tmp; }   // c[0]: the colour relaxed first
        }
        // the thread relaxes the same two cells in every sweep: their weights, 1/D and rhs stay in registers (16 doubles),
        // a relaxation reads the six neighbours from shared memory and nothing else (was 14 LDS.64 per relaxation: the
        // half-sweeps of a 1024-cell level were bound by shared-memory wavefronts, not by the barrier)
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
        // level constants and the neighbours' addresses in registers; the six neighbours are loaded before the first FMA
        // (the compiler otherwise re-reads nx and the z-stride from the kernel parameters -- indexed constant loads -- and
        // chains load -> FMA -> load inside every half-sweep)
        const int nx = L.nx, zs = L.zs;
        double* const ph = s.phi;
        auto relax = [&](int q) {
            if (c[q] < 0) return;                  // warps without a cell of this level go straight to the barrier
            double* const x = ph + cc[q];
            const double a0 = x[-1], a1 = x[1], a2 = x[-nx], a3 = x[nx], a4 = x[-zs], a5 = x[zs];
            double v = w[q][0] * a0;
            v = fma(w[q][1], a1, v);
            v = fma(w[q][2], a2, v);
            v = fma(w[q][3], a3, v);
            v = fma(w[q][4], a4, v);
            v = fma(w[q][5], a5, v);
            *x = di[q] * (rh[q] + v);
        };
        if (nt <= 32) {
            if (threadIdx.x < 32)
                for (int sw = 0; sw < nsweeps; ++sw) {
#pragma unroll
                    for (int q = 0; q < 2; ++q) {
                        relax(q);
                        __syncwarp();
                    }
                }
            __syncthreads();
            return;
        }
        for (int sw = 0; sw < nsweeps; ++sw) {
#pragma unroll
            for (int q = 0; q < 2; ++q) {
                relax(q);
                __syncthreads();
            }
        }
        return;
    }
    for (int sw = 0; sw < nsweeps; ++sw)
        for (int c2 = 0; c2 < 2; ++c2) {
            const int colour = (first + c2) & 1;
            for (int t = threadIdx.x; t < nt; t += blockDim.x) {
                int m = t % hx, j = (t / hx) % L.ny, k = t / (hx * L.ny);
                int i = 2 * m + ((colour + j + k) & 1);
                if (i < L.nx) {
                    int c = i + L.nx * j + L.nxy * k;
                    s.phi[c] = s.dinv[c] * (s.rhs[c] + tail_nb_sum(s, L, c));
                }
            }
            __syncthreads();
        }
}

__device__ __forceinline__ double tail_residual_at(const TailSmem& s, const TailLevel& L, int c)
{
    return s.rhs[c] + tail_nb_sum(s, L, c) - s.phi[c] / s.dinv[c];
}

// levels lev[0] .. lev[g.nl-1], by one CTA, in shared memory
#ifdef VMG_TAIL_TIMING
__device__ long long vmg_tail_clock[64];
#define TAIL_MARK(i) do { if (threadIdx.x == 0) vmg_tail_clock[i] = clock64(); } while (0)
#else
#define TAIL_MARK(i) do { } while (0)
#endif

// off: offset of this CTA's problem in a batched launch (vmg_create_batch), 0 for a single solve
__device__ __forceinline__ void coarse_tail_body(const TailArgs& g, const long long off)
{
    TAIL_MARK(0);
    extern __shared__ __align__(16) double tail_smem[];
    const int tid = threadIdx.x, nth = blockDim.x;

    // ---- stage in: zero everything (guards), then copy coefficients of every level, rhs (and phi) of the first ----
    {
        const TailLevel& B = g.lev[g.nl - 1];
        int total = B.off + tail_level_doubles(B.n, B.guard);
        for (int t = tid; t < total; t += nth) tail_smem[t] = 0.0;
    }
    __syncthreads();
    for (int l = 0; l < g.nl; ++l) {
        const TailLevel& L = g.lev[l];
        TailSmem s(tail_smem, L);
        for (int t = tid; t < L.n; t += nth) {
            const long long c = off + cell_at(L.G, t % L.nx, (t / L.nx) % L.ny, t / L.nxy);
            s.dinv[t] = L.dinv[c]; s.wx[t] = L.wx[c]; s.wy[t] = L.wy[c]; s.wz[t] = L.wz[c];
            if (l == 0) { s.rhs[t] = L.rhs[c]; if (g.whole) s.phi[t] = L.phi[c]; }
        }
    }
    __syncthreads();
    TAIL_MARK(1);

    // ---- down-stroke ----
    for (int l = 0; l + 1 < g.nl; ++l) {
        const TailLevel& L = g.lev[l];
        const TailLevel& C = g.lev[l + 1];
        TailSmem s(tail_smem, L), c(tail_smem, C);
        tail_smooth(s, L, g.nu1);
        TAIL_MARK(2 + 2 * l);
        for (int t = tid; t < C.n; t += nth) {     // residual + restriction (same order as residual_restrict_kernel)
            int I = t % C.nx, J = (t / C.nx) % C.ny, K = t / (C.nx * C.ny);
            double acc = 0.0;
            for (int r = 0; r < g.sz; ++r)
                for (int q = 0; q < 2; ++q) {
                    int cc = (2 * I) + L.nx * (2 * J + q) + L.nx * L.ny * (g.sz * K + r);
                    acc += tail_residual_at(s, L, cc) + tail_residual_at(s, L, cc + 1);
                }
            c.rhs[t] = acc / (4.0 * g.sz);
            c.phi[t] = 0.0;
        }
        __syncthreads();
        TAIL_MARK(3 + 2 * l);
    }
    // ---- bottom: fixed number of sweeps from zero (R11) ----
    {
        const TailLevel& B = g.lev[g.nl - 1];
        TailSmem s(tail_smem, B);
        if (g.nl == 1 && g.whole) {                 // single-level hierarchy: the bottom solve is the cycle (C4)
            for (int t = tid; t < B.n; t += nth) s.phi[t] = 0.0;
            __syncthreads();
        }
        if (g.S && !g.sym && !(g.nl == 1 && g.whole)) {   // the sweeps from zero as a matrix (bottom_matrix_kernel)
            const double* S = g.S + off;
            double acc = 0.0;
            if (tid < B.n)
                for (int j = 0; j < B.n; ++j) acc = fma(S[tid * B.n + j], s.rhs[j], acc);
            if (tid < B.n) s.phi[tid] = acc;
            __syncthreads();
        }
        else if (!g.sym) tail_smooth(s, B, g.nbottom);
        else { tail_smooth(s, B, g.nbottom / 2, 0); tail_smooth(s, B, g.nbottom - g.nbottom / 2, 1); }
    }
    TAIL_MARK(20);
    // ---- up-stroke ----
    for (int l = g.nl - 2; l >= 0; --l) {
        const TailLevel& L = g.lev[l];
        const TailLevel& C = g.lev[l + 1];
        TailSmem s(tail_smem, L), c(tail_smem, C);
        for (int t = tid; t < L.n; t += nth) {     // prolongation + correction (R9: piecewise constant, or trilinear)
            int i = t % L.nx, j = (t / L.nx) % L.ny, k = t / L.nxy;
            if (g.prolong) {
                const int par[3] = {i >> 1, j >> 1, g.sz == 2 ? (k >> 1) : k}, fine[3] = {i, j, k}, n[3] = {C.nx, C.ny, C.nz};
                s.phi[t] += trilinear_value(par, fine, n, g.sz, g.bc, c.phi, at_tail, &C);
            } else
                s.phi[t] += c.phi[(i >> 1) + C.nx * ((j >> 1) + C.ny * (g.sz == 2 ? (k >> 1) : k))];
        }
        __syncthreads();
        TAIL_MARK(21 + 2 * l);
        tail_smooth(s, L, g.nu2, g.sym);
        TAIL_MARK(22 + 2 * l);
    }
    // ---- stage out ----
    {
        const TailLevel& L = g.lev[0];
        TailSmem s(tail_smem, L);
        double m = 0.0;
        bool nan = false;
        for (int t = tid; t < L.n; t += nth) {
            L.phi[off + cell_at(L.G, t % L.nx, (t / L.nx) % L.ny, t / L.nxy)] = s.phi[t];
            if (g.whole && g.norm_out) {
                double x = fabs(tail_residual_at(s, L, t));
                nan |= (x != x);
                m = fmax(m, x);
            }
        }
        if (g.whole && g.norm_out) {
            if (nan) m = __longlong_as_double(0x7ff8000000000000ll);
            block_max_to_global(m, g.norm_out + off);   // (a batched launch: this problem's scalar)
        }
    }
    TAIL_MARK(40);
}


// NT: the largest CTA this instantiation is launched with (512 leaves the compiler 128 registers per thread)
template <int NT>
__global__ void __launch_bounds__(NT, 1) coarse_tail_kernel(TailArgs g)
{
    grid_dependency_wait();
    coarse_tail_body(g, (long long)blockIdx.x * g.pstride);
}

}  // namespace vmg
