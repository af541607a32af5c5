// vmg_pcg.cuh -- kernels of the MG-preconditioned conjugate gradients (vmg_solve_pcg in vmg_api.cu).
//
//     r = b - A x;  z = M^-1 r;  p = z;  rho = <r, z>
//     repeat:  q = A p;  alpha = rho / <p, q>;  x += alpha p;  r -= alpha q;  ||r||_inf
//              z = M^-1 r;  rho' = <r, z>;  p = z + (rho'/rho) p;  rho = rho'
//
// M^-1 is one symmetric V-cycle from a zero guess (option "symmetric": post-smoothing black -> red), which runs on
// the level-0 arrays: r lives in the level's rhs array, z in its phi array.  x, p, q are three more arrays in the
// internal layout (their pad elements stay zero, so the element-wise kernels simply run over the whole allocation).
// The scalars never visit the host: dot products are reduced in two deterministic stages (per-CTA partial sums in
// a fixed order, then one CTA over the partials) and the second stage forms alpha / beta in place; only the
// residual norm is read back, once per iteration, for the exit rules.
#pragma once
#include "vmg_kernels.cuh"

namespace vmg {

constexpr int kPcgThreads = 256;
enum { PCG_RHO = 0, PCG_PQ = 1, PCG_ALPHA = 2, PCG_BETA = 3 };   // slots of the scalar array
enum { PCG_MODE_RHO0 = 0, PCG_MODE_ALPHA = 1, PCG_MODE_BETA = 2 };

__device__ __forceinline__ double block_sum(double v)
{
    __shared__ double warp_sum[32];
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) warp_sum[w] = v;
    __syncthreads();
    double s = 0.0;
    if (w == 0) {
        const int nw = (blockDim.x + 31) >> 5;
        s = lane < nw ? warp_sum[lane] : 0.0;
        for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    }
    return s;   // valid in thread 0
}

// q = A p on every cell (A p = D p - sum w p_nb, D = 1/dinv), partial[blockIdx.x] = sum over the CTA of p*q
__global__ void pcg_apply_dot_kernel(LevelView L, const double* __restrict__ p, double* __restrict__ q, double* __restrict__ partial)
{
    grid_dependency_wait();
    const Geom& G = L.G;
    const long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    const long long nt = (long long)G.ne * G.ny * G.nz;
    double acc = 0.0;
    if (t < nt) {
        int m, j, k;
        unflatten_pair(G, t, m, j, k);
        const long long row = G.plane * k + (long long)G.pitch * j;
#pragma unroll
        for (int par = 0; par < 2; ++par) {
            if (2 * m + par >= G.nx) break;
            long long c, xm;
            pair_addr(G, row, m, par, c, xm);
            const double v = p[c] / L.dinv[c] - nb_sum(L, p, c, xm);
            q[c] = v;
            acc = fma(p[c], v, acc);
        }
    }
    const double s = block_sum(acc);
    if (threadIdx.x == 0) partial[blockIdx.x] = s;
}

// partial[blockIdx.x] = sum over the CTA of u*v (whole allocation; pads are zero)
__global__ void pcg_dot_kernel(const double* __restrict__ u, const double* __restrict__ v, long long n, double* __restrict__ partial)
{
    grid_dependency_wait();
    double acc = 0.0;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x)
        acc = fma(u[t], v[t], acc);
    const double s = block_sum(acc);
    if (threadIdx.x == 0) partial[blockIdx.x] = s;
}

// one CTA: the sum of the partials in a fixed order, then the scalar the iteration needs next
__global__ void pcg_reduce_kernel(const double* __restrict__ partial, int n, int mode, double* __restrict__ scal)
{
    grid_dependency_wait();
    double acc = 0.0;
    for (int t = threadIdx.x; t < n; t += blockDim.x) acc += partial[t];
    const double s = block_sum(acc);
    if (threadIdx.x == 0) {
        if (mode == PCG_MODE_RHO0) scal[PCG_RHO] = s;
        else if (mode == PCG_MODE_ALPHA) { scal[PCG_PQ] = s; scal[PCG_ALPHA] = scal[PCG_RHO] / s; }
        else { scal[PCG_BETA] = s / scal[PCG_RHO]; scal[PCG_RHO] = s; }
    }
}

// x += alpha p;  r -= alpha q;  ||r||_inf into *norm_out (zeroed by the caller)
__global__ void pcg_update_kernel(double* __restrict__ x, double* __restrict__ r, const double* __restrict__ p,
                                  const double* __restrict__ q, long long n, const double* __restrict__ scal,
                                  unsigned long long* norm_out)
{
    grid_dependency_wait();
    const double alpha = scal[PCG_ALPHA];
    double mx = 0.0;
    bool nan = false;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
        x[t] = fma(alpha, p[t], x[t]);
        const double rv = fma(-alpha, q[t], r[t]);
        r[t] = rv;
        const double a = fabs(rv);
        nan |= (a != a);
        mx = fmax(mx, a);
    }
    if (nan) mx = __longlong_as_double(0x7ff8000000000000ll);
    block_max_to_global(mx, norm_out);
}

// p = z + beta p   (first: p = z)
__global__ void pcg_direction_kernel(double* __restrict__ p, const double* __restrict__ z, long long n,
                                     const double* __restrict__ scal, int first)
{
    grid_dependency_wait();
    const double beta = first ? 0.0 : scal[PCG_BETA];
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x)
        p[t] = first ? z[t] : fma(beta, p[t], z[t]);
}

// r = b - A x in place of b (all cells), for the start of the iteration
__global__ void pcg_residual_inplace_kernel(LevelView L, const double* __restrict__ x, double* __restrict__ b)
{
    grid_dependency_wait();
    const Geom& G = L.G;
    const long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    const long long nt = (long long)G.ne * G.ny * G.nz;
    if (t >= nt) return;
    int m, j, k;
    unflatten_pair(G, t, m, j, k);
    const long long row = G.plane * k + (long long)G.pitch * j;
#pragma unroll
    for (int par = 0; par < 2; ++par) {
        if (2 * m + par >= G.nx) break;
        long long c, xm;
        pair_addr(G, row, m, par, c, xm);
        b[c] = residual_at(L, x, b, c, xm);
    }
}

}  // namespace vmg
