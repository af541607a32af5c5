// vmg_block.cuh -- S2 (+S3, S4, S6 fused): temporally blocked red-black Gauss-Seidel (north_star (2): "staging 3D
// tiles through ... shared memory with coalesced, vectorised fp64 loads and temporal blocking of several smoothing
// sweeps per tile").
//
// One pass applies S consecutive colour half-sweeps (optionally preceded by prolongation+correction applied while
// loading, optionally followed by a residual stage that feeds the restriction or the infinity norm) while every
// array of the level is read from global memory ONCE and phi is written once.
//
// Decomposition ("2.5-D" blocking).  The x-y plane is cut into tiles of TX x TY cells.  A CTA streams a tile along
// z: plane zl is loaded (with a halo of 4 cells in x, H in y) into a ring of planes in shared memory, then stage s
// = 1..S advances plane zl-s from state s-1 to state s (state = number of half-sweeps applied).  Stage s on plane p
// needs plane p+1 at state s-1 (done by stage s-1 in the same iteration) and plane p-1 at state s or s-1 (its cells
// of the other colour are the same in both).  Cells on the rim of the loaded tile are never updated, so the region
// holding correct state-s values shrinks by one cell per stage; with H >= S the TX x TY interior is exact.  Plane
// zl-S then leaves the ring for phi_out.  Passes ping-pong between two phi arrays because tiles overlap.
// The (tile, z) space is cut into equal contiguous segments, one per CTA ("stream-K"), each paying H extra planes at
// both ends; out-of-domain cells are loaded as zeros (zero weights, zero 1/D), which keeps them at zero.
//
// Shared-memory layout.  Thread t owns the x-pair (2m, 2m+1) of row j, t = j*NXP + m, for every plane: it loads the
// pair with one 16-byte access per array and stores the two cells split by colour, K[colour][t], so that a
// half-sweep (which touches one colour of a plane) reads and writes unit-stride fp64 vectors: no bank conflicts.
// Neighbours of the active cell of pair t in the other-colour array: x-1, x+1 -> t-1+sel, t+sel (sel = 0 if the
// active cell is the even one), y-1, y+1 -> t-NXP, t+NXP, z-1, z+1 -> t in the rings of planes p-1, p+1.
// In one iteration a thread's active cell is the same for all stages ((j + zl) parity), so every thread works in
// every stage.
//
// The arithmetic of one relaxation is the same expression, in the same order, as smooth_colour_kernel: results are
// bitwise identical to the one-launch-per-colour path.
#pragma once
#include "vmg_kernels.cuh"

namespace vmg {

enum { BT_NONE = 0, BT_RESTRICT = 1, BT_NORM = 2 };

struct BlockArgs {
    const double *wx, *wy, *wz, *dinv, *rhs;   // level arrays, internal stencil form (cell 0)
    const double* phi_in;
    double* phi_out;
    int nx, ny, nz;
    long long nxy;
    int colour0;                   // colour of the first half-sweep of this pass (0 = red = (i+j+k) even)
    int ntx, nty;                  // tiles in x and y
    int nzseg;                     // z-segments per tile; gridDim.x = ntx * nty * nzseg, tile index fastest
    const double* e;               // PROLONG: coarse correction (cnx x cny x cnz)
    double *crhs, *cphi;           // BT_RESTRICT: coarse right-hand side (written), coarse phi (zeroed)
    int cnx, cny;
    unsigned long long* norm_out;  // BT_NORM
};

template <int S, int TAIL, int NXT, int NYT>
struct BlockCfg {
    static constexpr int H = S + (TAIL ? 1 : 0);          // halo in y and z
    static constexpr int HX = 4;                          // halo in x (kept 32-byte aligned)
    static constexpr int TX = NXT - 2 * HX, TY = NYT - 2 * H;
    static constexpr int NXP = NXT / 2, NP = NXP * NYT;   // pairs per row, pairs per plane
    static constexpr int NT = (NP + 31) / 32 * 32;        // threads
    static constexpr int RP = S + 2 + (TAIL ? 1 : 0);     // phi ring
    static constexpr int RC = S + (TAIL ? 1 : 0);         // rhs, dinv, wx, wy rings
    static constexpr int RZ = RC + 1;                     // wz ring
    static constexpr int PLANE = 2 * NP;                  // doubles per plane of one array (two colours)
    static constexpr size_t SMEM = (size_t)((RP + 4 * RC + RZ) * PLANE + (TAIL == BT_RESTRICT ? NP : 0)) * sizeof(double);
    static_assert(H >= S && HX >= H && TX > 0 && TY > 0 && TX % 2 == 0 && TY % 2 == 0, "tile");
};

__device__ __forceinline__ double2 ldg2(const double* p) { return __ldg(reinterpret_cast<const double2*>(p)); }

template <int S, int TAIL, bool PROLONG, int NXT, int NYT>
__global__ void __launch_bounds__(BlockCfg<S, TAIL, NXT, NYT>::NT, 1) smooth_block_kernel(BlockArgs g)
{
    using C = BlockCfg<S, TAIL, NXT, NYT>;
    constexpr int H = C::H, NXP = C::NXP, NP = C::NP, RP = C::RP, RC = C::RC, RZ = C::RZ, PLANE = C::PLANE;
    extern __shared__ __align__(16) double blk_smem[];
    double* const s_phi = blk_smem;
    double* const s_rhs = s_phi + RP * PLANE;
    double* const s_dinv = s_rhs + RC * PLANE;
    double* const s_wx = s_dinv + RC * PLANE;
    double* const s_wy = s_wx + RC * PLANE;
    double* const s_wz = s_wy + RC * PLANE;
    double* const s_scr = s_wz + RZ * PLANE;      // BT_RESTRICT only

    const int t = threadIdx.x;
    const bool live = t < NP;
    const int m = t % NXP, j = t / NXP;

    // finite garbage only: anything multiplied by a zero weight must not be NaN/Inf
    for (int q = t; q < (int)(C::SMEM / sizeof(double)); q += C::NT) blk_smem[q] = 0.0;
    __syncthreads();

    // CTA -> (tile, z-segment), tile index fastest: the CTAs that run at the same time are x-y neighbours marching
    // through the same z-range in step, so that the tile halos they share are fetched from HBM once and hit in L2
    // for the others.  Segments are cut at even z so that restriction pairs stay together.
    const int ntiles = g.ntx * g.nty;
    double nrm = 0.0;
    bool nrm_nan = false;
    {
        const int tile = (int)(blockIdx.x % ntiles), seg = (int)(blockIdx.x / ntiles);
        const int za = (int)((long long)(g.nz / 2) * seg / g.nzseg) * 2;
        const int zb = seg == g.nzseg - 1 ? g.nz : (int)((long long)(g.nz / 2) * (seg + 1) / g.nzseg) * 2;
        const int tx = tile % g.ntx, ty = tile / g.ntx;
        const int gx = tx * C::TX - C::HX + 2 * m, gy = ty * C::TY - H + j;
        const bool in_xy = live && gx >= 0 && gx < g.nx && gy >= 0 && gy < g.ny;
        const bool interior = in_xy && m >= C::HX / 2 && m < C::HX / 2 + C::TX / 2 && j >= H && j < H + C::TY;
        const bool row_ok = live && j >= 1 && j <= NYT - 2;
        const long long cbase = gx + (long long)g.nx * gy;
        const long long ebase = PROLONG ? (gx >> 1) + (long long)g.cnx * (gy >> 1) : 0;

        double2 r_phi, r_wz, r_rhs, r_dinv, r_wx, r_wy;
        auto issue = [&](int zq) {   // phi, wz of plane zq; rhs, dinv, wx, wy of plane zq - 1
            const double2 zero = make_double2(0.0, 0.0);
            r_phi = r_wz = r_rhs = r_dinv = r_wx = r_wy = zero;
            if (in_xy && zq >= 0 && zq < g.nz) {
                long long c = cbase + g.nxy * zq;
                r_phi = ldg2(g.phi_in + c);
                r_wz = ldg2(g.wz + c);
                if (PROLONG) {
                    double ev = __ldg(g.e + ebase + (long long)g.cnx * g.cny * (zq >> 1));
                    r_phi.x += ev; r_phi.y += ev;
                }
            }
            if (in_xy && zq - 1 >= 0 && zq - 1 < g.nz) {
                long long c = cbase + g.nxy * (zq - 1);
                r_rhs = ldg2(g.rhs + c);
                r_dinv = ldg2(g.dinv + c);
                r_wx = ldg2(g.wx + c);
                r_wy = ldg2(g.wy + c);
            }
        };

        const int z0 = za - H;
        issue(z0);
        double acc = 0.0;   // BT_RESTRICT: running sum of the children of one coarse cell (even rows of even planes)

        for (int zl = z0; zl <= zb + H - 1; ++zl) {
            const int it = zl - z0;
            // ---- fill: registers -> rings (colour split), then prefetch the next plane into registers ----
            if (live) {
                const int ke = (gy + zl) & 1;            // colour of the even cell of the pair in plane zl
                double* p = s_phi + (it % RP) * PLANE;
                p[ke * NP + t] = r_phi.x; p[(ke ^ 1) * NP + t] = r_phi.y;
                p = s_wz + (it % RZ) * PLANE;
                p[ke * NP + t] = r_wz.x; p[(ke ^ 1) * NP + t] = r_wz.y;
                const int kc = ke ^ 1;                   // ... in plane zl - 1
                const int sc = ((it + RC - 1) % RC) * PLANE;
                s_rhs[sc + kc * NP + t] = r_rhs.x;   s_rhs[sc + (kc ^ 1) * NP + t] = r_rhs.y;
                s_dinv[sc + kc * NP + t] = r_dinv.x; s_dinv[sc + (kc ^ 1) * NP + t] = r_dinv.y;
                s_wx[sc + kc * NP + t] = r_wx.x;     s_wx[sc + (kc ^ 1) * NP + t] = r_wx.y;
                s_wy[sc + kc * NP + t] = r_wy.x;     s_wy[sc + (kc ^ 1) * NP + t] = r_wy.y;
            }
            if (zl + 1 <= zb + H - 1) issue(zl + 1);
            __syncthreads();

            // ---- stages: half-sweep s on plane zl - s ----
#pragma unroll
            for (int s = 1; s <= S; ++s) {
                const int p = zl - s;
                const int kc = (g.colour0 + s - 1) & 1;          // colour relaxed by this stage
                const int sel = (kc + gy + p) & 1;               // 0: the even cell of the pair is active
                const bool ok = row_ok && (sel ? m < NXP - 1 : m > 0);
                if (ok) {
                    const double* po = s_phi + ((it + RP - s) % RP) * PLANE + (kc ^ 1) * NP;     // other colour, plane p
                    const double* pm = s_phi + ((it + 2 * RP - s - 1) % RP) * PLANE + (kc ^ 1) * NP;   // plane p-1
                    const double* pp = s_phi + ((it + RP - s + 1) % RP) * PLANE + (kc ^ 1) * NP;   // plane p+1
                    const int sc = ((it + 2 * RC - s) % RC) * PLANE;   // coefficient plane q sits in slot (q - z0) % RC
                    const double* wzl = s_wz + ((it + RZ - s) % RZ) * PLANE + kc * NP;
                    const double* wzh = s_wz + ((it + RZ - s + 1) % RZ) * PLANE + (kc ^ 1) * NP;
                    double v = s_wx[sc + kc * NP + t] * po[t - 1 + sel];
                    v = fma(s_wx[sc + (kc ^ 1) * NP + t + sel], po[t + sel], v);
                    v = fma(s_wy[sc + kc * NP + t], po[t - NXP], v);
                    v = fma(s_wy[sc + (kc ^ 1) * NP + t + NXP], po[t + NXP], v);
                    v = fma(wzl[t], pm[t], v);
                    v = fma(wzh[t], pp[t], v);
                    s_phi[((it + RP - s) % RP) * PLANE + kc * NP + t] = s_dinv[sc + kc * NP + t] * (s_rhs[sc + kc * NP + t] + v);
                }
                __syncthreads();
            }

            // ---- plane zl - S is final: write it back ----
            {
                const int p = zl - S;
                if (interior && p >= za && p < zb) {
                    const int ke = (gy + p) & 1;
                    const double* q = s_phi + ((it + RP - S) % RP) * PLANE;
                    double2 o = make_double2(q[ke * NP + t], q[(ke ^ 1) * NP + t]);
                    *reinterpret_cast<double2*>(g.phi_out + cbase + g.nxy * p) = o;
                }
            }

            // ---- residual stage on plane zl - S - 1 (all its neighbours are final) ----
            if (TAIL != BT_NONE) {
                const int p = zl - S - 1;
                const bool on = p >= za && p < zb;     // uniform over the CTA
                double re = 0.0, ro = 0.0;
                if (on && interior) {
                    const int ke = (gy + p) & 1;
                    const int sp = ((it + RP - S - 1) % RP) * PLANE, sm = ((it + 2 * RP - S - 2) % RP) * PLANE,
                              sq = ((it + RP - S) % RP) * PLANE;
                    const int sc = ((it + 2 * RC - S - 1) % RC) * PLANE;
                    const int zlo = ((it + RZ - S - 1) % RZ) * PLANE, zhi = ((it + RZ - S) % RZ) * PLANE;
#pragma unroll
                    for (int sel = 0; sel < 2; ++sel) {
                        const int kc = ke ^ sel;                 // colour of this cell
                        const double* po = s_phi + sp + (kc ^ 1) * NP;
                        double v = s_wx[sc + kc * NP + t] * po[t - 1 + sel];
                        v = fma(s_wx[sc + (kc ^ 1) * NP + t + sel], po[t + sel], v);
                        v = fma(s_wy[sc + kc * NP + t], po[t - NXP], v);
                        v = fma(s_wy[sc + (kc ^ 1) * NP + t + NXP], po[t + NXP], v);
                        v = fma(s_wz[zlo + kc * NP + t], s_phi[sm + (kc ^ 1) * NP + t], v);
                        v = fma(s_wz[zhi + (kc ^ 1) * NP + t], s_phi[sq + (kc ^ 1) * NP + t], v);
                        double r = s_rhs[sc + kc * NP + t] + v - s_phi[sp + kc * NP + t] / s_dinv[sc + kc * NP + t];
                        if (sel == 0) re = r; else ro = r;
                    }
                    if (TAIL == BT_NORM) {
                        double a = fabs(re), b = fabs(ro);
                        nrm_nan |= (a != a) | (b != b);
                        nrm = fmax(nrm, fmax(a, b));
                    }
                }
                if (TAIL == BT_RESTRICT) {
                    // children are summed as in residual_restrict_kernel: per (z, y) the x-pair first, then accumulated
                    const double pair = re + ro;
                    if (on && live && (gy & 1)) s_scr[t] = pair;
                    __syncthreads();
                    if (on && interior && !(gy & 1)) {
                        acc += pair;
                        acc += s_scr[t + NXP];
                        if (p & 1) {
                            long long cc = (gx >> 1) + (long long)g.cnx * ((gy >> 1) + (long long)g.cny * (p >> 1));
                            g.crhs[cc] = acc / 8.0;
                            g.cphi[cc] = 0.0;
                            acc = 0.0;
                        }
                    }
                } else {
                    __syncthreads();   // the next fill overwrites plane zl - S - 2, which this stage has just read
                }
            }
        }
    }

    if (TAIL == BT_NORM) {
        if (nrm_nan) nrm = __longlong_as_double(0x7ff8000000000000ll);
        block_max_to_global(nrm, g.norm_out);
    }
}

}  // namespace vmg
