// vmg_block2.cuh -- S2 (+S3, S4, S6 fused): temporally blocked red-black Gauss-Seidel, second design
// (north_star (2): "staging 3D tiles through ... shared memory with coalesced, vectorised fp64 loads and temporal
// blocking of several smoothing sweeps per tile").
//
// One pass applies S consecutive colour half-sweeps (optionally preceded by prolongation+correction applied while
// loading, optionally followed by a residual stage that feeds the restriction or the infinity norm) while every
// array of the level is read from global memory ONCE and phi is written once.
//
// Decomposition ("2.5-D" blocking).  The x-y plane is cut into tiles of TX x TY cells, z into segments; one CTA
// per (tile, segment), tile index fastest, so that the CTAs resident at the same time are x-y neighbours marching
// through the same z-range in step and the tile halos they share are fetched from HBM once and hit in L2 for the
// others.  A CTA streams its tile along z: in iteration zl, stage s = 1..S advances plane zl-s from state s-1 to
// state s (state = number of half-sweeps applied).  Stage s on plane p needs plane p+1 at state s-1 (done by stage
// s-1 in the same iteration) and plane p-1 at state s or s-1 (its cells of the other colour are the same in both).
// Cells on the rim of the loaded tile are never updated, so the region holding correct state-s values shrinks by
// one cell per stage; with a halo of H >= S cells the TX x TY interior is exact.  Passes ping-pong between two phi
// arrays because tiles overlap.  Out-of-domain cells are loaded as zeros (zero weights, zero 1/D): they stay zero.
//
// Where the data lives (what the first design got wrong: every operand of every relaxation came from shared
// memory, 15 LDS.64 + 1 STS.64 = 32 shared-memory wavefronts per warp-update, more than the 128 B/clk port can
// feed at the HBM rate).  Thread t owns a 2 x 2 patch: the x-pair (2m, 2m+1) of rows 2jj and 2jj+1, t = jj*NXP + m,
// in every plane, and keeps in REGISTERS what only it ever reads: its own phi columns (planes zl .. zl-S-1: the
// z-neighbours, the pair-mate and the y-neighbour inside the patch of the cells it relaxes) and its own wz columns.
// Shared memory holds, for the S planes in flight, what OTHER threads read: phi (x- and y-neighbour outside the
// patch) and rhs, 1/D, wx, wy, split by x-parity and by row parity so that a half-sweep (which touches one
// x-parity per row) reads and writes unit-stride fp64 vectors without bank conflicts.  One relaxation = 8 LDS.64 +
// 1 STS.64.  Global loads are register-staged one plane ahead (24 x 8-byte loads per thread per plane: the level arrays
// are stored x-parity split), so data
// in flight costs no shared memory; a 2 x 2 patch per thread halves the thread count, which leaves each thread the
// ~170 registers that the rings, the staged loads and the residual stage need without spilling.
//
// No index arithmetic at run time.  Tiles start at even x, y, z offsets plus the halo, so the x-parity of the cell
// a thread relaxes in row r of iteration n is (colour0 + r + n + 1) & 1 for every thread of the grid: colour0 is a
// template parameter and the z-loop is unrolled by the period R of the register rings (even), which makes every
// register index, every parity and every shared-memory offset (relative to one base per stage) a compile-time
// constant: no selects, no ring rotation moves.
//
// The arithmetic of one relaxation / residual is the same expression, in the same order, as smooth_colour_kernel /
// residual_at: results are bitwise identical to the one-launch-per-step path.
#pragma once
#include "vmg_kernels.cuh"

namespace vmg {

enum { BT_NONE = 0, BT_RESTRICT = 1, BT_NORM = 2 };

struct BlockArgs {
    const double *wx, *wy, *wz, *dinv, *rhs;   // level arrays, internal stencil form (cell 0)
    const double* phi_in;
    double* phi_out;
    Geom G, CG;                    // layout of the level arrays and of the next coarser level's (vmg_kernels.cuh)
    int colour0;                   // colour of the first half-sweep of this pass (0 = red = (i+j+k) even)
    int ntx, nty;                  // tiles in x and y
    int nzseg;                     // z-segments per tile; gridDim.x = ntx * nty * nzseg, tile index fastest
    const double* e;               // PROLONG: coarse correction (cnx x cny x cnz)
    double *crhs, *cphi;           // BT_RESTRICT: coarse right-hand side (written), coarse phi (zeroed)
    unsigned long long* norm_out;  // BT_NORM
};


template <int S, int TAIL, int NXT, int NYT>
struct BlockCfg {
    // halo in y and z; with a residual stage S+1, rounded up to even so that a thread's two rows are the two
    // y-children of one coarse cell
    static constexpr int H = TAIL ? (S + 2) / 2 * 2 : S;
    static constexpr int HX = 4;                          // halo in x (kept 32-byte aligned)
    static constexpr int TX = NXT - 2 * HX, TY = NYT - 2 * H;
    static constexpr int NXP = NXT / 2, NPH = NXP * (NYT / 2);   // x-pairs per row, 2x2 patches per plane (= threads)
    static constexpr int NT = (NPH + 31) / 32 * 32;
    static constexpr int RS = S + (TAIL ? 1 : 0);         // shared-memory ring: planes zl-1 .. zl-RS
    static constexpr int R = (S + 4) / 2 * 2;             // register rings: planes zl .. zl-S-2 (S+3 planes), period even
    static constexpr int ARR = 4 * NPH;                   // one array of one plane: [x-parity][row parity][NPH]
    static constexpr int SLOT = 5 * ARR;                  // phi, rhs, dinv, wx, wy
    static constexpr size_t SMEM = (size_t)(RS * SLOT) * sizeof(double);
    static_assert(H >= S + (TAIL ? 1 : 0) && HX >= H && TX > 0 && TY > 0 &&
                      TX % 2 == 0 && TY % 2 == 0 && NYT % 2 == 0 && R >= S + 3 && R % 2 == 0, "tile");
};

__device__ __forceinline__ void prefetch_l2(const double* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
constexpr int kBlkPrefetch = 2;   // planes ahead of the register-staged loads

template <int S, int TAIL, bool PROLONG, int C0, int NXT, int NYT>
__global__ void __launch_bounds__(BlockCfg<S, TAIL, NXT, NYT>::NT, 1) smooth_block_kernel(BlockArgs g)
{
    using C = BlockCfg<S, TAIL, NXT, NYT>;
    constexpr int H = C::H, NXP = C::NXP, NPH = C::NPH, RS = C::RS, R = C::R, SLOT = C::SLOT;
    constexpr int A_PHI = 0, A_RHS = C::ARR, A_DINV = 2 * C::ARR, A_WX = 3 * C::ARR, A_WY = 4 * C::ARR;
    constexpr int XB = 2 * NPH;                     // offset of the odd-x block inside an array
    extern __shared__ __align__(16) double blk_smem[];

    const bool live = threadIdx.x < NPH;
    const int t = live ? threadIdx.x : 0;          // idle lanes of the last warp shadow thread 0 (and commit nothing)
    const int m = t % NXP, jj = t / NXP;

    // planes before the first loaded one: zero weights and zero 1/D keep them at zero (finite)
    for (int q = threadIdx.x; q < RS * SLOT; q += C::NT) blk_smem[q] = 0.0;

    // CTA -> (tile, z-segment), tile index fastest; segments are cut at even z (restriction pairs stay together)
    const int ntiles = g.ntx * g.nty;
    const int tile = (int)(blockIdx.x % ntiles), seg = (int)(blockIdx.x / ntiles);
    const int za = (int)((long long)(g.G.nz / 2) * seg / g.nzseg) * 2;
    const int zb = seg == g.nzseg - 1 ? g.G.nz : (int)((long long)(g.G.nz / 2) * (seg + 1) / g.nzseg) * 2;
    const int tx = tile % g.ntx, ty = tile / g.ntx;
    const int gx = tx * C::TX - C::HX + 2 * m, gy0 = ty * C::TY - H + 2 * jj;      // rows gy0 and gy0 + 1
    const bool in_x = live && gx >= 0 && gx < g.G.nx;
    const bool in_r[2] = {in_x && gy0 >= 0 && gy0 < g.G.ny, in_x && gy0 + 1 >= 0 && gy0 + 1 < g.G.ny};
    const bool int_x = m >= C::HX / 2 && m < C::HX / 2 + C::TX / 2;
    const bool interior[2] = {in_r[0] && int_x && 2 * jj >= H && 2 * jj < H + C::TY,
                              in_r[1] && int_x && 2 * jj + 1 >= H && 2 * jj + 1 < H + C::TY};
    // rows 0 and NYT-1 and the first / last column of the tile are rim: never relaxed.  ok[r][sg]: row r, x-parity sg
    const bool ok[2][2] = {{live && jj >= 1 && m > 0, live && jj >= 1 && m < NXP - 1},
                           {live && jj <= NYT / 2 - 2 && m > 0, live && jj <= NYT / 2 - 2 && m < NXP - 1}};
    // the x-pair's even cell in row gy0 of plane 0 (internal layout); its odd cell is `odd` further on
    const long long cbase = (long long)g.G.pitch * gy0 + (gx >> 1);
    const int odd = g.G.hp;

    // register rings [row][slot]: even-x / odd-x phi and wz of this thread's pair; plane z0 + n lives in slot n % R
    double pe[2][R], po[2][R], we[2][R], wo[2][R];
#pragma unroll
    for (int r = 0; r < 2; ++r)
#pragma unroll
        for (int k = 0; k < R; ++k) pe[r][k] = po[r][k] = we[r][k] = wo[r][k] = 0.0;
    int sl[RS];                                    // sl[k]: offset of the slot holding plane zl - 1 - k, + t
#pragma unroll
    for (int k = 0; k < RS; ++k) sl[k] = k * SLOT + t;

    // loads in flight: phi, wz (and the coarse correction) of plane zq; rhs, 1/D, wx, wy of plane zq - 1
    double2 r_phi[2], r_wz[2], r_rhs[2], r_dinv[2], r_wx[2], r_wy[2];
    double r_e[2] = {0.0, 0.0};
    auto ld2 = [&](const double* p, long long c) { return make_double2(__ldg(p + c), __ldg(p + c + odd)); };
    auto issue = [&](int zq) {
        // pull the planes kBlkPrefetch further on from HBM into L2 now (one request per 32-byte sector): all CTAs march
        // in step, so their loads come in bursts; with the DRAM latency taken early the staged loads below hit L2
        if (!(m & 3) && zq + kBlkPrefetch < g.G.nz && zq + kBlkPrefetch > 0) {
#pragma unroll
            for (int r = 0; r < 2; ++r)
                if (in_r[r]) {
                    const long long c = cbase + r * g.G.pitch + g.G.plane * (zq + kBlkPrefetch);
#pragma unroll
                    for (int o = 0; o < 2; ++o) {
                        const long long d = c + o * odd;
                        prefetch_l2(g.phi_in + d); prefetch_l2(g.wz + d);
                        prefetch_l2(g.rhs + d - g.G.plane); prefetch_l2(g.dinv + d - g.G.plane);
                        prefetch_l2(g.wx + d - g.G.plane); prefetch_l2(g.wy + d - g.G.plane);
                    }
                }
        }
        const double2 zero = make_double2(0.0, 0.0);
#pragma unroll
        for (int r = 0; r < 2; ++r) {
            r_phi[r] = r_wz[r] = r_rhs[r] = r_dinv[r] = r_wx[r] = r_wy[r] = zero;
            r_e[r] = 0.0;
            if (in_r[r] && zq >= 0 && zq < g.G.nz) {
                const long long c = cbase + r * g.G.pitch + g.G.plane * zq;
                r_phi[r] = ld2(g.phi_in, c);
                r_wz[r] = ld2(g.wz, c);
                if (PROLONG) r_e[r] = __ldg(g.e + cell_at(g.CG, gx >> 1, (gy0 + r) >> 1, zq >> 1));
            }
            if (in_r[r] && zq - 1 >= 0 && zq - 1 < g.G.nz) {
                const long long c = cbase + r * g.G.pitch + g.G.plane * (zq - 1);
                r_rhs[r] = ld2(g.rhs, c);
                r_dinv[r] = ld2(g.dinv, c);
                r_wx[r] = ld2(g.wx, c);
                r_wy[r] = ld2(g.wy, c);
            }
        }
    };

    const int z0 = za - H, z1 = zb + H - 1;
    issue(z0);
#pragma unroll
    for (int r = 0; r < 2; ++r) {                  // plane z0 -> slot 0
        if (PROLONG) { r_phi[r].x += r_e[r]; r_phi[r].y += r_e[r]; }
        pe[r][0] = r_phi[r].x; po[r][0] = r_phi[r].y; we[r][0] = r_wz[r].x; wo[r][0] = r_wz[r].y;
    }
    issue(z0 + 1);
    __syncthreads();

    double nrm = 0.0;
    bool nrm_nan = false;
    double acc = 0.0;    // BT_RESTRICT: running sum over the children of one coarse cell (even plane, then odd plane)

    for (int zbase = z0; zbase <= z1; zbase += R) {
#pragma unroll
        for (int u = 0; u < R; ++u) {
            const int zl = zbase + u;              // iteration n = zl - z0, n % R == u
            if (zl > z1) break;                    // uniform

            // ---- stages: half-sweep s on plane zl - s (ring slot (u-s) % R, shared slot sl[s-1]); rim threads compute
            // and discard.  Row r relaxes its cell of x-parity sg = (C0 + r + u + 1) & 1. ----
#pragma unroll
            for (int s = 1; s <= S; ++s) {
                const int c = ((u - s) % R + R) % R, cu = ((u - s + 1) % R + R) % R, cd = ((u - s - 1) % R + R) % R;
                double* P = blk_smem + sl[s - 1];
                double nv[2];
#pragma unroll
                for (int r = 0; r < 2; ++r) {
                    const int sg = (C0 + r + u + 1) & 1;
                    const int oA = sg * XB + r * NPH;                                   // active cell
                    const double mate = sg ? pe[r][c] : po[r][c];
                    const double zup = sg ? po[r][cu] : pe[r][cu], zdn = sg ? po[r][cd] : pe[r][cd];
                    const double wzl = sg ? wo[r][c] : we[r][c], wzh = sg ? wo[r][cu] : we[r][cu];
                    const double yin = sg ? po[1 - r][c] : pe[1 - r][c];
                    const double xo = P[A_PHI + (sg ? r * NPH + 1 : XB + r * NPH - 1)];   // x-neighbour outside the pair
                    const double yo = P[A_PHI + sg * XB + (r ? NXP : NPH - NXP)];        // y-neighbour outside the patch
                    const double xm = sg ? mate : xo, xp = sg ? xo : mate;
                    const double ym = r ? yin : yo, yp = r ? yo : yin;
                    double v = P[A_WX + oA] * xm;
                    v = fma(P[A_WX + (sg ? r * NPH + 1 : XB + r * NPH)], xp, v);
                    v = fma(P[A_WY + oA], ym, v);
                    v = fma(P[A_WY + sg * XB + (r ? NXP : NPH)], yp, v);
                    v = fma(wzl, zdn, v);
                    v = fma(wzh, zup, v);
                    nv[r] = P[A_DINV + oA] * (P[A_RHS + oA] + v);
                }
#pragma unroll
                for (int r = 0; r < 2; ++r) {
                    const int sg = (C0 + r + u + 1) & 1;
                    if (ok[r][sg]) {
                        if (sg) po[r][c] = nv[r]; else pe[r][c] = nv[r];
                        P[A_PHI + sg * XB + r * NPH] = nv[r];
                    }
                }

                // ---- residual stage on plane zl - S - 1 (shared slot sl[S]); all its neighbours are final: plane
                // zl - S in this thread's registers (just relaxed), the others since the previous iteration ----
                if (TAIL != BT_NONE && s == S) {
                    const int pr = zl - S - 1;
                    if (pr >= za && pr < zb && interior[0]) {     // interior rows come in pairs (H, TY, ny are even)
                        const int k = ((u - S - 1) % R + R) % R, ku = ((u - S) % R + R) % R, kd = ((u - S - 2) % R + R) % R;
                        const double* Q = blk_smem + sl[RS - 1];
                        double res[2][2];                    // [row][x-parity]
#pragma unroll
                        for (int r = 0; r < 2; ++r)
#pragma unroll
                            for (int e = 0; e < 2; ++e) {
                                const int o = e * XB + r * NPH;
                                const double ce = e ? po[r][k] : pe[r][k], mate = e ? pe[r][k] : po[r][k];
                                const double xo = Q[A_PHI + (e ? r * NPH + 1 : XB + r * NPH - 1)];
                                const double yo = Q[A_PHI + e * XB + (r ? NXP : NPH - NXP)];
                                const double yin = e ? po[1 - r][k] : pe[1 - r][k];
                                const double xm = e ? mate : xo, xp = e ? xo : mate;
                                const double ym = r ? yin : yo, yp = r ? yo : yin;
                                double v = Q[A_WX + o] * xm;
                                v = fma(Q[A_WX + (e ? r * NPH + 1 : XB + r * NPH)], xp, v);
                                v = fma(Q[A_WY + o], ym, v);
                                v = fma(Q[A_WY + e * XB + (r ? NXP : NPH)], yp, v);
                                v = fma(e ? wo[r][k] : we[r][k], e ? po[r][kd] : pe[r][kd], v);
                                v = fma(e ? wo[r][ku] : we[r][ku], e ? po[r][ku] : pe[r][ku], v);
                                res[r][e] = Q[A_RHS + o] + v - ce / Q[A_DINV + o];
                            }
                        if (TAIL == BT_NORM) {
#pragma unroll
                            for (int r = 0; r < 2; ++r)
#pragma unroll
                                for (int e = 0; e < 2; ++e) {
                                    const double a = fabs(res[r][e]);
                                    nrm_nan |= (a != a);
                                    nrm = fmax(nrm, a);
                                }
                        }
                        if (TAIL == BT_RESTRICT) {
                            // S3: children summed as in residual_restrict_kernel: per (z, y) the x-pair first, then accumulated
                            acc += res[0][0] + res[0][1];
                            acc += res[1][0] + res[1][1];
                            if (pr & 1) {
                                const long long cc = cell_at(g.CG, gx >> 1, gy0 >> 1, pr >> 1);
                                g.crhs[cc] = acc / 8.0;
                                g.cphi[cc] = 0.0;
                                acc = 0.0;
                            }
                        }
                    }
                }
                __syncthreads();
            }

            // ---- plane zl - S is final: write it back from registers ----
            {
                const int p = zl - S, c = ((u - S) % R + R) % R;
                if (p >= za && p < zb) {
#pragma unroll
                    for (int r = 0; r < 2; ++r)
                        if (interior[r]) {
                            double* q = g.phi_out + cbase + r * g.G.pitch + g.G.plane * p;
                            q[0] = pe[r][c]; q[odd] = po[r][c];
                        }
                }
            }
            // ---- plane zl (still untouched, ring slot u) and its coefficients replace plane zl - RS in shared memory ----
            if (live) {
                double* F = blk_smem + sl[RS - 1];
#pragma unroll
                for (int r = 0; r < 2; ++r) {
                    const int o0 = r * NPH, o1 = XB + r * NPH;
                    F[A_PHI + o0] = pe[r][u];     F[A_PHI + o1] = po[r][u];
                    F[A_RHS + o0] = r_rhs[r].x;   F[A_RHS + o1] = r_rhs[r].y;
                    F[A_DINV + o0] = r_dinv[r].x; F[A_DINV + o1] = r_dinv[r].y;
                    F[A_WX + o0] = r_wx[r].x;     F[A_WX + o1] = r_wx[r].y;
                    F[A_WY + o0] = r_wy[r].x;     F[A_WY + o1] = r_wy[r].y;
                }
            }
            {
                const int freed = sl[RS - 1];
#pragma unroll
                for (int k = RS - 1; k > 0; --k) sl[k] = sl[k - 1];
                sl[0] = freed;
            }
            // ---- plane zl + 1 enters the register rings (slot (u+1) % R held plane zl + 1 - R, no longer needed) ----
#pragma unroll
            for (int r = 0; r < 2; ++r) {
                const int n1 = (u + 1) % R;
                if (PROLONG) { r_phi[r].x += r_e[r]; r_phi[r].y += r_e[r]; }   // S4: phi += P e; r_e = 0 off-domain
                pe[r][n1] = r_phi[r].x; po[r][n1] = r_phi[r].y; we[r][n1] = r_wz[r].x; wo[r][n1] = r_wz[r].y;
            }
            if (zl < z1) issue(zl + 2);
            __syncthreads();
        }
    }

    if (TAIL == BT_NORM) {
        if (nrm_nan) nrm = __longlong_as_double(0x7ff8000000000000ll);
        block_max_to_global(nrm, g.norm_out);
    }
}

}  // namespace vmg
