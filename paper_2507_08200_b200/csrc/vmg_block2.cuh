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
// feed at the HBM rate).  Thread t owns the x-pair (2m, 2m+1) of row j, t = j*NXP + m, in every plane, and keeps
// in REGISTERS what only it ever reads: its own phi column (planes zl .. zl-S-1: the z-neighbours and the
// pair-mate of the cell it relaxes) and its own wz column.  Shared memory holds, for the S planes in flight, what
// OTHER threads read: phi (x-neighbour outside the pair, y-neighbours) and rhs, 1/D, wx, wy, split by x-parity so
// that a half-sweep (which touches one parity per row) reads and writes unit-stride fp64 vectors without bank
// conflicts.  One relaxation = 9 LDS.64 + 1 STS.64.  Global loads are register-staged one plane ahead
// (6 x 16-byte loads per thread per plane), so data in flight costs no shared memory.
//
// Register rings are indexed by ROLE, not by x-parity: in plane q the cell relaxed at odd stages has x-parity
// (colour0 + gy + q) & 1 ("role A"), the other is "role B".  Roles swap parity from plane to plane, so the
// z-neighbours and the pair-mate of a role-A cell are role-B cells: every register index is a compile-time
// constant.  In one iteration the active cell has the same x-parity sigma in all stages, sigma flips per iteration.
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
    static constexpr int RS = S + (TAIL ? 1 : 0);         // shared-memory ring: planes zl-1 .. zl-RS
    static constexpr int RPSI = S + 2 + (TAIL ? 1 : 0);   // register ring of phi: planes zl .. zl-RPSI+1
    static constexpr int RWZ = S + 1 + (TAIL ? 1 : 0);    // register ring of wz:  planes zl .. zl-RWZ+1
    static constexpr int SLOT = 10 * NP;                  // doubles per slot: phi, rhs, dinv, wx, wy, each [2][NP]
    static constexpr size_t SMEM = (size_t)(RS * SLOT + (TAIL == BT_RESTRICT ? NP : 0)) * sizeof(double);
    static_assert(H >= S && HX >= H && TX > 0 && TY > 0 && TX % 2 == 0 && TY % 2 == 0, "tile");
};

__device__ __forceinline__ double2 ldg2(const double* p) { return __ldg(reinterpret_cast<const double2*>(p)); }
__device__ __forceinline__ void prefetch_l2(const double* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
constexpr int kBlkPrefetch = 2;   // planes ahead of the register-staged loads

template <int S, int TAIL, bool PROLONG, int NXT, int NYT>
__global__ void __launch_bounds__(BlockCfg<S, TAIL, NXT, NYT>::NT, 1) smooth_block_kernel(BlockArgs g)
{
    using C = BlockCfg<S, TAIL, NXT, NYT>;
    constexpr int H = C::H, NXP = C::NXP, NP = C::NP, RS = C::RS, RPSI = C::RPSI, RWZ = C::RWZ, SLOT = C::SLOT;
    constexpr int A_PHI = 0, A_RHS = 2 * NP, A_DINV = 4 * NP, A_WX = 6 * NP, A_WY = 8 * NP;   // arrays inside a slot
    extern __shared__ __align__(16) double blk_smem[];
    double* const s_scr = blk_smem + RS * SLOT;   // BT_RESTRICT only

    const int t = threadIdx.x;
    const bool live = t < NP;
    const int m = t % NXP, j = t / NXP;

    // planes before the first loaded one: zero weights and zero 1/D keep them at zero (finite)
    for (int q = t; q < (int)(C::SMEM / sizeof(double)); q += C::NT) blk_smem[q] = 0.0;

    // CTA -> (tile, z-segment), tile index fastest; segments are cut at even z (restriction pairs stay together)
    const int ntiles = g.ntx * g.nty;
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
    const int par0 = g.colour0 + gy;   // + plane index: x-parity of the role-A cell of that plane

    // register rings, index k <-> plane zl - k (role A / role B values of this thread's pair)
    double pa[RPSI], pb[RPSI], wa[RWZ], wb[RWZ];
#pragma unroll
    for (int k = 0; k < RPSI; ++k) pa[k] = pb[k] = 0.0;
#pragma unroll
    for (int k = 0; k < RWZ; ++k) wa[k] = wb[k] = 0.0;
    int sl[RS];                                    // sl[k]: offset of the slot holding plane zl - 1 - k
#pragma unroll
    for (int k = 0; k < RS; ++k) sl[k] = k * SLOT;

    // loads in flight: phi, wz (and the coarse correction) of plane zq; rhs, 1/D, wx, wy of plane zq - 1
    double2 r_phi, r_wz, r_rhs, r_dinv, r_wx, r_wy;
    double r_e = 0.0;
    auto issue = [&](int zq) {
        // pull the planes kBlkPrefetch further on from HBM into L2 now: all CTAs march in step, so their loads come
        // in bursts; with the DRAM latency taken early the register-staged loads below are L2 hits
        if (in_xy && zq + kBlkPrefetch < g.nz && zq + kBlkPrefetch > 0) {
            const long long c = cbase + g.nxy * (zq + kBlkPrefetch);
            prefetch_l2(g.phi_in + c); prefetch_l2(g.wz + c);
            prefetch_l2(g.rhs + c - g.nxy); prefetch_l2(g.dinv + c - g.nxy);
            prefetch_l2(g.wx + c - g.nxy); prefetch_l2(g.wy + c - g.nxy);
        }
        const double2 zero = make_double2(0.0, 0.0);
        r_phi = r_wz = r_rhs = r_dinv = r_wx = r_wy = zero;
        r_e = 0.0;
        if (in_xy && zq >= 0 && zq < g.nz) {
            const long long c = cbase + g.nxy * zq;
            r_phi = ldg2(g.phi_in + c);
            r_wz = ldg2(g.wz + c);
            if (PROLONG) r_e = __ldg(g.e + ebase + (long long)g.cnx * g.cny * (zq >> 1));
        }
        if (in_xy && zq - 1 >= 0 && zq - 1 < g.nz) {
            const long long c = cbase + g.nxy * (zq - 1);
            r_rhs = ldg2(g.rhs + c);
            r_dinv = ldg2(g.dinv + c);
            r_wx = ldg2(g.wx + c);
            r_wy = ldg2(g.wy + c);
        }
    };
    // rings move one plane on; the loaded phi, wz of plane zq become index 0 (pA = x-parity of its role-A cell)
    auto insert = [&](int pA) {
#pragma unroll
        for (int k = RPSI - 1; k > 0; --k) { pa[k] = pa[k - 1]; pb[k] = pb[k - 1]; }
#pragma unroll
        for (int k = RWZ - 1; k > 0; --k) { wa[k] = wa[k - 1]; wb[k] = wb[k - 1]; }
        if (PROLONG) { r_phi.x += r_e; r_phi.y += r_e; }   // S4: phi += P e (piecewise constant); r_e = 0 off-domain
        pa[0] = pA ? r_phi.y : r_phi.x; pb[0] = pA ? r_phi.x : r_phi.y;
        wa[0] = pA ? r_wz.y : r_wz.x;   wb[0] = pA ? r_wz.x : r_wz.y;
    };

    const int z0 = za - H, z1 = zb + H - 1;
    issue(z0);
    insert((par0 + z0) & 1);
    issue(z0 + 1);
    __syncthreads();

    double nrm = 0.0;
    bool nrm_nan = false;
    double acc = 0.0;    // BT_RESTRICT: running sum over the children of one coarse cell (even rows, even..odd plane)
    double pair = 0.0;

    for (int zl = z0; zl <= z1; ++zl) {
        const int sigma = (par0 + zl - 1) & 1;             // x-parity of the cells relaxed in this iteration
        const int offA = sigma * NP + t;                   // active cell (also: its wx_lo, wy_lo, rhs, 1/D)
        const int offX = sigma ? t + 1 : NP + t - 1;       // its x-neighbour outside the pair
        const int offW = sigma ? t + 1 : NP + t;           // wx of its high-x face
        const bool ok = row_ok && (sigma ? m < NXP - 1 : m > 0);

        // ---- stages: half-sweep s on plane zl - s (ring index s, slot sl[s-1]) ----
#pragma unroll
        for (int s = 1; s <= S; ++s) {
            if (ok) {
                double* P = blk_smem + sl[s - 1];
                double mate, zup, zdn, wzl, wzh;
                if (s & 1) { mate = pb[s]; zup = pb[s - 1]; zdn = pb[s + 1]; wzl = wa[s]; wzh = wb[s - 1]; }
                else       { mate = pa[s]; zup = pa[s - 1]; zdn = pa[s + 1]; wzl = wb[s]; wzh = wa[s - 1]; }
                const double xo = P[A_PHI + offX];
                const double xm = sigma ? mate : xo, xp = sigma ? xo : mate;
                double v = P[A_WX + offA] * xm;
                v = fma(P[A_WX + offW], xp, v);
                v = fma(P[A_WY + offA], P[A_PHI + offA - NXP], v);
                v = fma(P[A_WY + offA + NXP], P[A_PHI + offA + NXP], v);
                v = fma(wzl, zdn, v);
                v = fma(wzh, zup, v);
                const double nv = P[A_DINV + offA] * (P[A_RHS + offA] + v);
                if (s & 1) pa[s] = nv; else pb[s] = nv;
                P[A_PHI + offA] = nv;
            }

            // ---- residual stage on plane zl - S - 1 (ring index S+1, slot sl[S]); all its neighbours are final:
            // plane zl - S in this thread's registers (just relaxed), the others since the previous iteration ----
            if (TAIL != BT_NONE && s == S) {
                const int pr = zl - S - 1;
                const bool on = pr >= za && pr < zb;     // uniform over the CTA
                double res[2] = {0.0, 0.0};              // even-x cell, odd-x cell
                if (on && interior) {
                    constexpr int K = S + 1;             // ring index of plane pr
                    const double* P = blk_smem + sl[RS - 1];
                    // x-parity of the role-A cell of ring index k is sigma ^ ((k-1)&1)
                    const int pK = sigma ^ ((K - 1) & 1);
                    const double ce[2] = {pK ? pb[K] : pa[K], pK ? pa[K] : pb[K]};                           // plane pr
                    const double cu[2] = {pK ? pa[K - 1] : pb[K - 1], pK ? pb[K - 1] : pa[K - 1]};           // plane pr+1
                    const double cd[2] = {pK ? pa[K + 1] : pb[K + 1], pK ? pb[K + 1] : pa[K + 1]};           // plane pr-1
                    const double wl[2] = {pK ? wb[K] : wa[K], pK ? wa[K] : wb[K]};                           // wz of plane pr
                    const double wh[2] = {pK ? wa[K - 1] : wb[K - 1], pK ? wb[K - 1] : wa[K - 1]};           // wz of plane pr+1
#pragma unroll
                    for (int e = 0; e < 2; ++e) {
                        const int oA = e * NP + t;
                        const double xo = P[A_PHI + (e ? t + 1 : NP + t - 1)];
                        const double xm = e ? ce[0] : xo, xp = e ? xo : ce[1];
                        double v = P[A_WX + oA] * xm;
                        v = fma(P[A_WX + (e ? t + 1 : NP + t)], xp, v);
                        v = fma(P[A_WY + oA], P[A_PHI + oA - NXP], v);
                        v = fma(P[A_WY + oA + NXP], P[A_PHI + oA + NXP], v);
                        v = fma(wl[e], cd[e], v);
                        v = fma(wh[e], cu[e], v);
                        res[e] = P[A_RHS + oA] + v - ce[e] / P[A_DINV + oA];
                    }
                    if (TAIL == BT_NORM) {
                        const double a = fabs(res[0]), b = fabs(res[1]);
                        nrm_nan |= (a != a) | (b != b);
                        nrm = fmax(nrm, fmax(a, b));
                    }
                }
                if (TAIL == BT_RESTRICT) {
                    pair = res[0] + res[1];
                    if (on && live && (gy & 1)) s_scr[t] = pair;   // odd rows hand their x-pair sum to the row below
                }
            }
            __syncthreads();
        }

        // ---- plane zl - S is final: write it back from registers ----
        {
            const int p = zl - S;
            if (interior && p >= za && p < zb) {
                const int pS = sigma ^ ((S - 1) & 1);
                const double2 o = make_double2(pS ? pb[S] : pa[S], pS ? pa[S] : pb[S]);
                *reinterpret_cast<double2*>(g.phi_out + cbase + g.nxy * p) = o;
            }
        }
        // ---- S3: children are summed as in residual_restrict_kernel: per (z, y) the x-pair first, then accumulated ----
        if (TAIL == BT_RESTRICT) {
            const int pr = zl - S - 1;
            if (pr >= za && pr < zb && interior && !(gy & 1)) {
                acc += pair;
                acc += s_scr[t + NXP];
                if (pr & 1) {
                    const long long cc = (gx >> 1) + (long long)g.cnx * ((gy >> 1) + (long long)g.cny * (pr >> 1));
                    g.crhs[cc] = acc / 8.0;
                    g.cphi[cc] = 0.0;
                    acc = 0.0;
                }
            }
        }
        // ---- plane zl (still untouched, ring index 0) and its coefficients replace plane zl - RS in shared memory ----
        if (live) {
            double* F = blk_smem + sl[RS - 1];
            const int p0 = sigma ^ 1;                     // x-parity of the role-A cell of plane zl
            F[A_PHI + t] = p0 ? pb[0] : pa[0];   F[A_PHI + NP + t] = p0 ? pa[0] : pb[0];
            F[A_RHS + t] = r_rhs.x;              F[A_RHS + NP + t] = r_rhs.y;
            F[A_DINV + t] = r_dinv.x;            F[A_DINV + NP + t] = r_dinv.y;
            F[A_WX + t] = r_wx.x;                F[A_WX + NP + t] = r_wx.y;
            F[A_WY + t] = r_wy.x;                F[A_WY + NP + t] = r_wy.y;
        }
        {
            const int freed = sl[RS - 1];
#pragma unroll
            for (int k = RS - 1; k > 0; --k) sl[k] = sl[k - 1];
            sl[0] = freed;
        }
        insert(sigma);                                    // plane zl + 1: its role-A parity is (par0 + zl + 1) & 1 = sigma
        if (zl < z1) issue(zl + 2);
        __syncthreads();
    }

    if (TAIL == BT_NORM) {
        if (nrm_nan) nrm = __longlong_as_double(0x7ff8000000000000ll);
        block_max_to_global(nrm, g.norm_out);
    }
}

}  // namespace vmg
