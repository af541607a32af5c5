// vmg_amr.cuh -- kernels of the two-level composite solve (vmg_amr_* in include/vmg.h, second half;
// PAPER.md:157-159 "composite multilevel multigrid solver", non-subcycled AMR levels).  Readings A1-A5 of DESIGN.md:
// refinement ratio 2, one or several separated box patches away from the boundary; across a coarse-fine face a two-point flux over 1.5 hf
// between the fine cell and the coarse field interpolated linearly in the tangential directions; the coarse cell takes
// the sum of the fine fluxes.
//
// How the pieces of the single-level library are used: the PATCH is an ordinary handle whose box faces are all
// "Dirichlet" faces with the boundary-face weight scaled by 1/3 -- 2 * (beta b / 3 hf^2) = beta b / (1.5 hf^2) is exactly
// the coarse-fine weight -- and whose value planes are rewritten from the coarse field before every fold (amr_ghost_kernel).
// Smoother, residual + restriction, norms and fold_bc of the patch are then the library's own kernels.  The COARSE BOX is
// an ordinary handle too: its V-cycle, run in place on phi_c with a right-hand side that differs from btilde_c only in and
// next to the patch, is the correction solver; the composite residual of its uncovered cells is the library's residual with
// the flux through a face of the patch replaced by the fine fluxes (amr_patch_rhs_kernel).
#pragma once
#include "vmg_kernels.cuh"

namespace vmg {

struct AmrGeom {
    Geom C, F, S;            // coarse box, fine patch, the patch's shadow on the coarse level (= level 1 of the patch handle)
    int lo[3], hi[3], nd;    // patch in coarse cells [lo, hi); active directions
};

__device__ __forceinline__ bool amr_covered(const AmrGeom& A, int i, int j, int k)
{
    return i >= A.lo[0] && i < A.hi[0] && j >= A.lo[1] && j < A.hi[1] && (A.nd < 3 || (k >= A.lo[2] && k < A.hi[2]));
}

// the two axes of the value plane of a face normal to d, lower axis first (include/vmg.h: x faces j + ny k, y faces
// i + nx k, z faces i + nx j)
__device__ __forceinline__ void amr_plane_axes(int d, int& u, int& v) { u = d == 0 ? 1 : 0; v = d == 2 ? 1 : 2; }

// A2: value planes of the patch's faces, g = phi_C + sum_t s_t (phi_{C+e_t} - phi_{C-e_t}) / 8.  grid (blocks, 2 nd).
struct AmrGhostArgs { AmrGeom A; const double* phic; double* plane[6]; };

__global__ void amr_ghost_kernel(AmrGhostArgs g)
{
    const AmrGeom& A = g.A;
    const int f = blockIdx.y, d = f >> 1, side = f & 1;
    int ua, va;
    amr_plane_axes(d, ua, va);
    const int m[3] = {A.F.nx, A.F.ny, A.F.nz};
    const long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t >= (long long)m[ua] * m[va]) return;
    int fi[3], c[3];
    fi[ua] = (int)(t % m[ua]); fi[va] = (int)(t / m[ua]); fi[d] = side ? m[d] - 1 : 0;
    for (int a = 0; a < 3; ++a) c[a] = a < A.nd ? A.lo[a] + fi[a] / 2 : 0;
    c[d] += side ? 1 : -1;                               // the coarse cell across the face
    double gv = g.phic[cell_at(A.C, c[0], c[1], c[2])];
    for (int a = 0; a < A.nd; ++a) {
        if (a == d) continue;
        int p[3] = {c[0], c[1], c[2]}, q[3] = {c[0], c[1], c[2]};
        p[a] += 1; q[a] -= 1;
        const double s = (fi[a] & 1) ? 1.0 : -1.0;       // the fine centre lies h/4 above (odd) or below (even) C's centre
        gv += s * (g.phic[cell_at(A.C, p[0], p[1], p[2])] - g.phic[cell_at(A.C, q[0], q[1], q[2])]) / 8.0;
    }
    g.plane[f][t] = gv;
}

// the coarse cells under the patch become the means of their children (A4); one thread per shadow cell.  The mean is
// also kept in old[] (shadow order): the coarse V-cycle runs in place on phi_c, and the correction the patch receives
// is the difference to this value (amr_prolong_add_kernel).
__global__ void amr_average_down_kernel(AmrGeom A, const double* __restrict__ phif, double* __restrict__ phic, double* __restrict__ old)
{
    const long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t >= A.S.n) return;
    int i, j, k;
    unflatten(A.S, t, i, j, k);
    const int ns = A.nd == 3 ? 2 : 1;
    double sum = 0.0;
    for (int s = 0; s < ns; ++s)
        for (int q = 0; q < 2; ++q)
            for (int p = 0; p < 2; ++p) sum += phif[cell_at(A.F, 2 * i + p, 2 * j + q, A.nd == 3 ? 2 * k + s : 0)];
    const double mean = sum / (A.nd == 3 ? 8.0 : 4.0);
    phic[cell_at(A.C, A.lo[0] + i, A.lo[1] + j, A.nd == 3 ? A.lo[2] + k : 0)] = mean;
    old[t] = mean;
}

// A5: the folded coarse right-hand side does not count under the patch: zero it there, ||.||_inf of the rest -> *norm
__global__ void amr_mask_norm_kernel(AmrGeom A, double* __restrict__ btc, unsigned long long* norm)
{
    const long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    double v = 0.0;
    if (t < A.C.n) {
        int i, j, k;
        unflatten(A.C, t, i, j, k);
        const long long c = cell_at(A.C, i, j, k);
        if (amr_covered(A, i, j, k)) btc[c] = 0.0;
        v = fabs(btc[c]);
        if (v != v) v = __longlong_as_double(0x7ff8000000000000ll);
    }
    if (norm) block_max_to_global(v, norm);      // NULL: only zero under this patch (more patches follow)
}

// A3 + A4: the right-hand side of the coarse V-cycle, which runs IN PLACE on phi_c (solution form): one V-cycle maps
// (phi, rhs) to phi + B (rhs - A phi), so with rhs' = R + A phi_c (R: the right-hand side of the correction equation of A4,
// A: the plain coarse operator) it returns phi_c + B R, the corrected field -- and rhs' differs from btilde_c only where R
// is not the plain residual: on the covered cells and on the cells that share a face with the patch.  This kernel rewrites
// exactly those entries every cycle (one thread per cell of the patch's bounding box grown by one cell); every other
// entry of rhs' is btilde_c, copied once per solve.
//   uncovered cell next to the patch:  rhs' = btilde + (the coarse flux through the shared face taken out, the fluxes of the
//                                      fine faces on it put in; weights: the patch handle's scaled boundary planes,
//                                      2 wb / 2^nd = beta b_f / (1.5 hf) * area_f / volume_C; g: the patch's value planes)
//   covered cell:                      rhs' = R + A phi_c,  R = mean of the children's residuals (rs, residual_restrict_kernel
//                                      of the patch)
// With this rhs' the library's own residual norm over the box (residual_norm_kernel on rhs') IS the composite norm of A5:
// rhs' - A phi is the composite residual on every uncovered cell and R on the covered ones, where |mean of the children's
// residuals| <= ||r_f||_inf, which A5 takes anyway.  That kernel skips the black cells after the first cycle (R12: the
// V-cycle's last half-sweep has just relaxed them) -- but the black cells next to the patch changed their right-hand side
// since, so this kernel adds the residual of EVERY cell next to the patch to *norm itself.
struct AmrResArgs {
    AmrGeom A; LevelView Lc;
    const double *phic, *btc, *rs, *phif;
    double* R;
    const double* gplane[6]; const double* wbf[6];
    double wscale;
    unsigned long long* norm;
};

__global__ void amr_patch_rhs_kernel(AmrResArgs g)
{
    const AmrGeom& A = g.A;
    const long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    int ext[3] = {1, 1, 1};
    for (int a = 0; a < A.nd; ++a) ext[a] = A.hi[a] - A.lo[a] + 2;
    double mx = 0.0;
    if (t < (long long)ext[0] * ext[1] * ext[2]) {
        int ci[3] = {0, 0, 0};
        ci[0] = (int)(t % ext[0]) + A.lo[0] - 1;
        ci[1] = (int)((t / ext[0]) % ext[1]) + A.lo[1] - 1;
        if (A.nd == 3) ci[2] = (int)(t / ((long long)ext[0] * ext[1])) + A.lo[2] - 1;
        long long c, xm;
        pair_addr(A.C, A.C.plane * ci[2] + (long long)A.C.pitch * ci[1], ci[0] >> 1, ci[0] & 1, c, xm);
        if (amr_covered(A, ci[0], ci[1], ci[2])) {
            const double rs = g.rs[cell_at(A.S, ci[0] - A.lo[0], ci[1] - A.lo[1], A.nd == 3 ? ci[2] - A.lo[2] : 0)];
            g.R[c] = rs + (g.phic[c] / g.Lc.dinv[c] - nb_sum(g.Lc, g.phic, c, xm));
        } else {
            const int m[3] = {A.F.nx, A.F.ny, A.F.nz};
            double corr = 0.0;
            bool touched = false;
            for (int f = 0; f < 2 * A.nd; ++f) {
                const int d = f >> 1, side = f & 1;
                int q[3] = {ci[0], ci[1], ci[2]};
                q[d] += side ? 1 : -1;
                if (!amr_covered(A, q[0], q[1], q[2])) continue;
                touched = true;
                // the coarse face weight and the covered neighbour, as nb_sum addresses them
                const long long nb = d == 0 ? (side ? xm + 1 : xm) : d == 1 ? (side ? c + A.C.pitch : c - A.C.pitch)
                                                                            : (side ? c + A.C.plane : c - A.C.plane);
                const double* warr = d == 0 ? g.Lc.wx : d == 1 ? g.Lc.wy : g.Lc.wz;
                const double wface = warr[side ? nb : c];
                corr += wface * (g.phic[c] - g.phic[nb]);              // take the coarse flux out ...
                int ua, va;
                amr_plane_axes(d, ua, va);
                const int ff = 2 * d + (1 - side), nt = A.nd - 1;
                int ta[2], u = 0;
                for (int a = 0; a < A.nd; ++a) if (a != d) ta[u++] = a;
                for (u = 0; u < (1 << nt); ++u) {                      // ... and put the fine fluxes in
                    int F[3] = {0, 0, 0};
                    F[d] = side ? 0 : m[d] - 1;
                    for (int a = 0; a < nt; ++a) F[ta[a]] = 2 * (ci[ta[a]] - A.lo[ta[a]]) + ((u >> a) & 1);
                    const long long pi = F[ua] + (long long)m[ua] * F[va];
                    corr -= g.wbf[ff][pi] * g.wscale * (g.gplane[ff][pi] - g.phif[cell_at(A.F, F[0], F[1], F[2])]);
                }
            }
            if (touched) {
                g.R[c] = g.btc[c] + corr;
                mx = fabs(residual_at(g.Lc, g.phic, g.btc, c, xm) + corr);
                if (mx != mx) mx = __longlong_as_double(0x7ff8000000000000ll);
            }
        }
    }
    block_max_to_global(mx, g.norm);
}

// phi_f += the correction of the parent (piecewise constant, R9) = its new value - the mean it held before the V-cycle
__global__ void amr_prolong_add_kernel(AmrGeom A, double* __restrict__ phif, const double* __restrict__ phic, const double* __restrict__ old)
{
    const long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t >= A.F.n) return;
    int i, j, k;
    unflatten(A.F, t, i, j, k);
    const int I = i / 2, J = j / 2, K = A.nd == 3 ? k / 2 : 0;
    const double e = phic[cell_at(A.C, A.lo[0] + I, A.lo[1] + J, A.nd == 3 ? A.lo[2] + K : 0)]
                   - old[I + (long long)A.S.nx * (J + (long long)A.S.ny * K)];
    phif[cell_at(A.F, i, j, k)] += e;
}

__global__ void amr_scale_kernel(double* __restrict__ v, long long n, double s)
{
    const long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t < n) v[t] *= s;
}

}  // namespace vmg
