// vmg_kernels.cuh -- baseline (one step per launch) kernels of libvmg.  fp64 throughout.
// These are the correctness baseline every fused / blocked kernel is diffed against, and they remain the
// path for levels and options the blocked kernels do not cover.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

namespace vmg {

constexpr int kThreads = 256;

__host__ __device__ inline long long cdiv(long long a, long long b) { return (a + b - 1) / b; }

// ------------------------------------------------------------------------------------------------
// S0. Coefficient averaging to the next coarser level (north_star (2) "coefficient averaging";
// reading R10: a = mean of children, b = mean of the fine faces lying on the coarse face).
// Public layouts on both sides.  NULL fine a means a == 0; NULL fine b means b == 1.
// ------------------------------------------------------------------------------------------------
__global__ void coarsen_a_kernel(const double* __restrict__ fa, double* __restrict__ ca,
                                 int cnx, int cny, int cnz, int sz)
{
    long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    long long n = (long long)cnx * cny * cnz;
    if (t >= n) return;
    int I = (int)(t % cnx), J = (int)((t / cnx) % cny), K = (int)(t / ((long long)cnx * cny));
    int fnx = 2 * cnx, fny = 2 * cny;
    double s = 0.0;
    if (fa)
        for (int r = 0; r < sz; ++r)
            for (int q = 0; q < 2; ++q)
                for (int p = 0; p < 2; ++p)
                    s += fa[(2 * I + p) + (long long)fnx * ((2 * J + q) + (long long)fny * (sz * K + r))];
    ca[t] = s / (4.0 * sz);
}

// dir: 0 = x faces, 1 = y faces, 2 = z faces.  (cnx, cny, cnz) are coarse CELL counts.
__global__ void coarsen_b_kernel(const double* __restrict__ fb, double* __restrict__ cb,
                                 int cnx, int cny, int cnz, int sz, int dir)
{
    int ex = cnx + (dir == 0), ey = cny + (dir == 1), ez = cnz + (dir == 2);
    long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    long long n = (long long)ex * ey * ez;
    if (t >= n) return;
    int I = (int)(t % ex), J = (int)((t / ex) % ey), K = (int)(t / ((long long)ex * ey));
    int fex = 2 * cnx + (dir == 0), fey = 2 * cny + (dir == 1);
    if (!fb) { cb[t] = 1.0; return; }
    double s = 0.0;
    if (dir == 0) {
        for (int r = 0; r < sz; ++r) for (int q = 0; q < 2; ++q)
            s += fb[(2 * I) + (long long)fex * ((2 * J + q) + (long long)fey * (sz * K + r))];
        cb[t] = s / (2.0 * sz);
    } else if (dir == 1) {
        for (int r = 0; r < sz; ++r) for (int p = 0; p < 2; ++p)
            s += fb[(2 * I + p) + (long long)fex * ((2 * J) + (long long)fey * (sz * K + r))];
        cb[t] = s / (2.0 * sz);
    } else {
        for (int q = 0; q < 2; ++q) for (int p = 0; p < 2; ++p)
            s += fb[(2 * I + p) + (long long)fex * ((2 * J + q) + (long long)fey * (2 * K))];
        cb[t] = s / 4.0;
    }
}

// ------------------------------------------------------------------------------------------------
// Internal stencil form of one level from its raw coefficients (C1 of DESIGN.md).
// ------------------------------------------------------------------------------------------------
struct StencilBuildArgs {
    const double *a, *bx, *by, *bz;      // raw, public layout (may be NULL)
    double *wx, *wy, *wz, *dbase;        // padded cell arrays
    double* wb[6];                       // boundary planes
    int nx, ny, nz, three_d;
    double alpha, cx, cy, cz;            // cx = beta/hx^2 ...
};

__global__ void build_stencil_kernel(StencilBuildArgs g)
{
    long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    long long n = (long long)g.nx * g.ny * g.nz;
    if (t >= n) return;
    int i = (int)(t % g.nx), j = (int)((t / g.nx) % g.ny), k = (int)(t / ((long long)g.nx * g.ny));
    long long nxy = (long long)g.nx * g.ny;
    double bxl = g.bx ? g.bx[i + (long long)(g.nx + 1) * (j + (long long)g.ny * k)] : 1.0;
    double bxh = g.bx ? g.bx[i + 1 + (long long)(g.nx + 1) * (j + (long long)g.ny * k)] : 1.0;
    double byl = g.by ? g.by[i + (long long)g.nx * (j + (long long)(g.ny + 1) * k)] : 1.0;
    double byh = g.by ? g.by[i + (long long)g.nx * (j + 1 + (long long)(g.ny + 1) * k)] : 1.0;
    double wxl = g.cx * bxl, wxh = g.cx * bxh, wyl = g.cy * byl, wyh = g.cy * byh, wzl = 0.0, wzh = 0.0;
    if (g.three_d) {
        double bzl = g.bz ? g.bz[t] : 1.0;
        double bzh = g.bz ? g.bz[t + nxy] : 1.0;
        wzl = g.cz * bzl; wzh = g.cz * bzh;
    }
    if (i == 0)        { g.wb[0][j + (long long)g.ny * k] = wxl; wxl = 0.0; }
    if (i == g.nx - 1) { g.wb[1][j + (long long)g.ny * k] = wxh; wxh = 0.0; }
    if (j == 0)        { g.wb[2][i + (long long)g.nx * k] = wyl; wyl = 0.0; }
    if (j == g.ny - 1) { g.wb[3][i + (long long)g.nx * k] = wyh; wyh = 0.0; }
    if (g.three_d) {
        if (k == 0)        { g.wb[4][i + (long long)g.nx * j] = wzl; wzl = 0.0; }
        if (k == g.nz - 1) { g.wb[5][i + (long long)g.nx * j] = wzh; wzh = 0.0; }
    }
    g.wx[t] = wxl; g.wy[t] = wyl; g.wz[t] = wzl;
    double d = g.a ? g.alpha * g.a[t] : 0.0;
    d += wxl; d += wxh; d += wyl; d += wyh; d += wzl; d += wzh;
    g.dbase[t] = d;
}

struct DinvArgs {
    const double* dbase; double* dinv; const double* wb[6];
    int nx, ny, nz, three_d; int dirichlet[6];
};

__global__ void finalize_dinv_kernel(DinvArgs g)
{
    long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    long long n = (long long)g.nx * g.ny * g.nz;
    if (t >= n) return;
    int i = (int)(t % g.nx), j = (int)((t / g.nx) % g.ny), k = (int)(t / ((long long)g.nx * g.ny));
    double d = g.dbase[t];
    if (i == 0 && g.dirichlet[0])        d += 2.0 * g.wb[0][j + (long long)g.ny * k];
    if (i == g.nx - 1 && g.dirichlet[1]) d += 2.0 * g.wb[1][j + (long long)g.ny * k];
    if (j == 0 && g.dirichlet[2])        d += 2.0 * g.wb[2][i + (long long)g.nx * k];
    if (j == g.ny - 1 && g.dirichlet[3]) d += 2.0 * g.wb[3][i + (long long)g.nx * k];
    if (g.three_d) {
        if (k == 0 && g.dirichlet[4])        d += 2.0 * g.wb[4][i + (long long)g.nx * j];
        if (k == g.nz - 1 && g.dirichlet[5]) d += 2.0 * g.wb[5][i + (long long)g.nx * j];
    }
    g.dinv[t] = 1.0 / d;
}

// ------------------------------------------------------------------------------------------------
// S1. fold_bc: btilde = f + 2*w_b*g on Dirichlet-adjacent cells + w_b*h*q on Neumann-adjacent cells
// (w_b = beta*b/h^2 of the boundary face; R3, R5).  Level 0, once per solve.
// ------------------------------------------------------------------------------------------------
struct FoldArgs {
    const double* rhs; double* bt; const double* wb[6]; const double* val[6];
    int nx, ny, nz, three_d; int dirichlet[6]; double h[3];
};

__global__ void fold_bc_kernel(FoldArgs g)
{
    long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    long long n = (long long)g.nx * g.ny * g.nz;
    if (t >= n) return;
    int i = (int)(t % g.nx), j = (int)((t / g.nx) % g.ny), k = (int)(t / ((long long)g.nx * g.ny));
    double v = g.rhs[t];
    auto add = [&](int f, long long pl, double hd) {
        if (!g.val[f]) return;
        double w = g.wb[f][pl], q = g.val[f][pl];
        v += g.dirichlet[f] ? 2.0 * w * q : w * hd * q;
    };
    if (i == 0)        add(0, j + (long long)g.ny * k, g.h[0]);
    if (i == g.nx - 1) add(1, j + (long long)g.ny * k, g.h[0]);
    if (j == 0)        add(2, i + (long long)g.nx * k, g.h[1]);
    if (j == g.ny - 1) add(3, i + (long long)g.nx * k, g.h[1]);
    if (g.three_d) {
        if (k == 0)        add(4, i + (long long)g.nx * j, g.h[2]);
        if (k == g.nz - 1) add(5, i + (long long)g.nx * j, g.h[2]);
    }
    g.bt[t] = v;
}

// ------------------------------------------------------------------------------------------------
// The 7-point relaxation / operator in internal form.  All neighbour reads are in-bounds thanks to the
// zero pads and all out-of-domain neighbours carry a zero weight.
// ------------------------------------------------------------------------------------------------
struct LevelView {
    const double *wx, *wy, *wz, *dinv;
    int nx, ny, nz;
    long long nxy, n;
};

__device__ __forceinline__ double nb_sum(const LevelView& L, const double* __restrict__ phi, long long c)
{
    double s = L.wx[c] * phi[c - 1];
    s = fma(L.wx[c + 1], phi[c + 1], s);
    s = fma(L.wy[c], phi[c - L.nx], s);
    s = fma(L.wy[c + L.nx], phi[c + L.nx], s);
    s = fma(L.wz[c], phi[c - L.nxy], s);
    s = fma(L.wz[c + L.nxy], phi[c + L.nxy], s);
    return s;
}

// S2 (baseline). One colour half-sweep: phi_c <- (rhs_c + sum w phi_nb) / D_c for (i+j+k)%2 == colour.
// Planes [k0, k1) only (the L2 wavefront schedule launches it slab by slab).
__global__ void smooth_colour_kernel(LevelView L, double* __restrict__ phi, const double* __restrict__ rhs, int colour,
                                     int k0, int k1)
{
    int hx = (L.nx + 1) >> 1;
    long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    long long nt = (long long)hx * L.ny * (k1 - k0);
    if (t >= nt) return;
    int m = (int)(t % hx), j = (int)((t / hx) % L.ny), k = k0 + (int)(t / ((long long)hx * L.ny));
    int i = 2 * m + ((colour + j + k) & 1);
    if (i >= L.nx) return;
    long long c = i + (long long)L.nx * j + L.nxy * k;
    phi[c] = L.dinv[c] * (rhs[c] + nb_sum(L, phi, c));
}

// S4 + S2 fused (plain path).  The first colour half-sweep after a coarse-grid correction: a relaxation never reads
// the old value of the cell it overwrites, and all six neighbours of a cell of one colour have the other colour, so
// the correction phi += P e (piecewise constant, R9) is applied to the NEIGHBOURS on the fly and never stored: the
// cells of the other colour keep their uncorrected values in memory until the next half-sweep overwrites them.
// Valid when at least one full sweep follows (nu2 >= 1).  phi_nb + e is the very addition prolong_correct_kernel
// performs, so results are bitwise those of the two separate kernels.
__global__ void smooth_colour_prolong_kernel(LevelView L, double* __restrict__ phi, const double* __restrict__ rhs,
                                             const double* __restrict__ e, int colour, int sz)
{
    int hx = (L.nx + 1) >> 1;
    long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    long long nt = (long long)hx * L.ny * L.nz;
    if (t >= nt) return;
    int m = (int)(t % hx), j = (int)((t / hx) % L.ny), k = (int)(t / ((long long)hx * L.ny));
    int i = 2 * m + ((colour + j + k) & 1);
    if (i >= L.nx) return;
    long long c = i + (long long)L.nx * j + L.nxy * k;
    const int cnx = L.nx >> 1, cny = L.ny >> 1;
    const int K = sz == 2 ? (k >> 1) : k;
    auto ec = [&](int ii, int jj, int kk) { return e[(ii >> 1) + (long long)cnx * ((jj >> 1) + (long long)cny * kk)]; };
    // out-of-domain neighbours carry a zero weight; their (zero-pad) value is used uncorrected
    double xm = phi[c - 1], xp = phi[c + 1], ym = phi[c - L.nx], yp = phi[c + L.nx], zm = phi[c - L.nxy], zp = phi[c + L.nxy];
    if (i > 0) xm += ec(i - 1, j, K);
    if (i < L.nx - 1) xp += ec(i + 1, j, K);
    if (j > 0) ym += ec(i, j - 1, K);
    if (j < L.ny - 1) yp += ec(i, j + 1, K);
    if (sz == 2) {
        if (k > 0) zm += e[(i >> 1) + (long long)cnx * ((j >> 1) + (long long)cny * ((k - 1) >> 1))];
        if (k < L.nz - 1) zp += e[(i >> 1) + (long long)cnx * ((j >> 1) + (long long)cny * ((k + 1) >> 1))];
    }
    double s = L.wx[c] * xm;
    s = fma(L.wx[c + 1], xp, s);
    s = fma(L.wy[c], ym, s);
    s = fma(L.wy[c + L.nx], yp, s);
    s = fma(L.wz[c], zm, s);
    s = fma(L.wz[c + L.nxy], zp, s);
    phi[c] = L.dinv[c] * (rhs[c] + s);
}

// r = rhs - A phi, A phi = D phi - sum w phi_nb, D = 1/dinv.
__device__ __forceinline__ double residual_at(const LevelView& L, const double* __restrict__ phi,
                                              const double* __restrict__ rhs, long long c)
{
    return rhs[c] + nb_sum(L, phi, c) - phi[c] / L.dinv[c];
}

__global__ void residual_kernel(LevelView L, const double* __restrict__ phi, const double* __restrict__ rhs,
                                double* __restrict__ r)
{
    long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t >= L.n) return;
    r[t] = residual_at(L, phi, rhs, t);
}

// S3 (baseline). Fused residual + restriction: one thread per coarse cell; also zeroes the coarse phi.
// Coarse planes [K0, K1) only.
__global__ void residual_restrict_kernel(LevelView L, const double* __restrict__ phi, const double* __restrict__ rhs,
                                         double* __restrict__ crhs, double* __restrict__ cphi, int sz, int K0, int K1)
{
    int cnx = L.nx >> 1, cny = L.ny >> 1;
    long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    long long n = (long long)cnx * cny * (K1 - K0);
    if (t >= n) return;
    int I = (int)(t % cnx), J = (int)((t / cnx) % cny), K = K0 + (int)(t / ((long long)cnx * cny));
    t = I + (long long)cnx * (J + (long long)cny * K);
    double s = 0.0;
    for (int r = 0; r < sz; ++r)
        for (int q = 0; q < 2; ++q) {   // the x-pair first, then accumulated (the blocked kernel sums in this order too)
            long long c = (2 * I) + (long long)L.nx * (2 * J + q) + L.nxy * (sz * K + r);
            s += residual_at(L, phi, rhs, c) + residual_at(L, phi, rhs, c + 1);
        }
    crhs[t] = s / (4.0 * sz);
    if (cphi) cphi[t] = 0.0;
}

// S4 (baseline). Fused prolongation + correction (piecewise constant, R9): phi_f += e_c[i/2, j/2, k/2].
// Fine planes [k0, k1) only.
__global__ void prolong_correct_kernel(double* __restrict__ phi, const double* __restrict__ e,
                                       int nx, int ny, int sz, int k0, int k1)
{
    long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    long long n = (long long)nx * ny * (k1 - k0);
    if (t >= n) return;
    t += (long long)nx * ny * k0;
    int i = (int)(t % nx), j = (int)((t / nx) % ny), k = (int)(t / ((long long)nx * ny));
    int cnx = nx >> 1, cny = ny >> 1;
    phi[t] += e[(i >> 1) + (long long)cnx * ((j >> 1) + (long long)cny * (sz == 2 ? (k >> 1) : k))];
}

// ------------------------------------------------------------------------------------------------
// S6. Infinity norms: warp shuffle -> block reduce -> one atomicMax on the bit pattern (non-negative
// doubles order like unsigned 64-bit integers; a NaN's pattern is larger than every finite value, so
// it propagates to the host, which tests for it).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void block_max_to_global(double v, unsigned long long* out)
{
    unsigned long long b = (unsigned long long)__double_as_longlong(fabs(v));
    for (int o = 16; o > 0; o >>= 1) {
        unsigned long long other = __shfl_xor_sync(0xffffffffu, b, o);
        b = other > b ? other : b;
    }
    __shared__ unsigned long long warp_max[32];
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) warp_max[w] = b;
    __syncthreads();
    if (w == 0) {
        int nw = (blockDim.x + 31) >> 5;
        b = lane < nw ? warp_max[lane] : 0ull;
        for (int o = 16; o > 0; o >>= 1) {
            unsigned long long other = __shfl_xor_sync(0xffffffffu, b, o);
            b = other > b ? other : b;
        }
        if (lane == 0 && b != 0ull) atomicMax(out, b);
    }
}

__global__ void norm_inf_kernel(const double* __restrict__ v, long long n, unsigned long long* out)
{
    double m = 0.0;
    bool nan = false;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
        double x = fabs(v[t]);
        nan |= (x != x);
        m = fmax(m, x);
    }
    if (nan) m = __longlong_as_double(0x7ff8000000000000ll);
    block_max_to_global(m, out);
}

// planes [k0, k1) only; accumulates into *out with atomicMax (the caller zeroes it)
__global__ void residual_norm_kernel(LevelView L, const double* __restrict__ phi, const double* __restrict__ rhs,
                                     unsigned long long* out, int k0, int k1)
{
    double m = 0.0;
    bool nan = false;
    long long t1 = L.nxy * k1;
    for (long long t = L.nxy * k0 + blockIdx.x * (long long)blockDim.x + threadIdx.x; t < t1; t += (long long)gridDim.x * blockDim.x) {
        double x = fabs(residual_at(L, phi, rhs, t));
        nan |= (x != x);
        m = fmax(m, x);
    }
    if (nan) m = __longlong_as_double(0x7ff8000000000000ll);
    block_max_to_global(m, out);
}

}  // namespace vmg
