// vmg_block3.cuh -- S2 (+S3, S4, S6 fused): temporally blocked red-black Gauss-Seidel, third design: TMA-fed.
// (north_star (2): "staging 3D tiles through TMA or shared memory with coalesced, vectorised fp64 loads and temporal
// blocking of several smoothing sweeps per tile"; the linear solves are the paper's GPU obstacle.)
//
// Same decomposition and the same arithmetic as vmg_block2.cuh ("2.5-D" blocking: x-y tiles with a halo stream along
// z, stage s = 1..S advances plane zl-s by one colour half-sweep in iteration zl; thread = 2 x 2 patch whose own phi
// and wz columns live in register rings; bitwise the results of the one-launch-per-colour path).  What changed is how
// the data moves and how the threads wait for each other:
//
//  * The operands OTHER threads read (phi, wx, wy) arrive by TMA.  A level array in the x-parity split layout is a
//    legal 5-D tensor (m, row pair, row parity, x-parity, plane) -- every stride is a multiple of 16 bytes since a half
//    row is padded to 4 doubles (Geom::hp) -- and a box {NXP, NYT/2, 2, 2, 1} of it lands in shared memory as
//    [x-parity][row parity][patch], i.e. exactly the conflict-free layout the stages index with the thread number.
//    Out-of-domain parts of a box are zero-filled by the hardware (zero weights keep such cells at zero).  One elected
//    thread issues three cp.async.bulk.tensor per plane into a ring of NS slots, each slot with its own mbarrier
//    (complete_tx); a cp.async.bulk.prefetch.tensor pulls the planes two further on into L2.  No staging registers, no
//    STS to fill the ring.
//  * The operands only the owning thread reads (rhs, 1/D, wz) never needed to be shared: wz goes from global memory
//    straight into the register ring, rhs and 1/D into a thread-private ring (shared memory here; see PRIV).
//  * ONE barrier per plane instead of S+1: in iteration zl the stages work on S different planes; what stage s reads
//    from its neighbours was written by stage s-1 in iteration zl-1.  The barrier is split (mbarrier arrive by one lane
//    per warp after the last write of an iteration, try_wait before the first neighbour read of the next), so the
//    global stores, the private loads and the pull of the next plane sit between arrive and wait.
#pragma once
#include <cuda.h>
#include "vmg_kernels.cuh"
#include "vmg_block2.cuh"   // BT_NONE / BT_RESTRICT / BT_NORM

namespace vmg {

struct alignas(64) Block3Args {
    CUtensorMap tm_phi, tm_wx, tm_wy;     // 5-D views of phi_in, wx, wy (make_level_tensor_map in vmg_sched.cuh)
    const double *wz, *dinv, *rhs;        // thread-private operands, plain loads (cell 0, internal layout)
    double* phi_out;
    Geom G, CG;
    int colour0;                          // (unused by the kernel: the colour is a template parameter)
    int ntx, nty, nzseg;                  // tiles in x, y; z-segments per tile; gridDim.x = ntx*nty*nzseg, tile fastest
    const double* e;                      // PROLONG: coarse correction
    double *crhs, *cphi;                  // BT_RESTRICT
    unsigned long long* norm_out;         // BT_NORM
};

// ---- PTX: mbarrier, TMA, proxy fence ----
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* b, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* b, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* b)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* b, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}" ::"r"(smem_u32(b)), "r"(parity) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }

// box of the 5-D tensor at (m, row pair, 0, 0, plane) -> dst; completion (bytes) on bar
__device__ __forceinline__ void tma_load_5d(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1, int c4)
{
    asm volatile(
        "cp.async.bulk.tensor.5d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(0), "r"(0), "r"(c4) : "memory");
}
__device__ __forceinline__ void tma_prefetch_5d(const CUtensorMap* map, int c0, int c1, int c4)
{
    asm volatile("cp.async.bulk.prefetch.tensor.5d.L2.global [%0, {%1, %2, %3, %4, %5}];"
                 ::"l"(map), "r"(c0), "r"(c1), "r"(0), "r"(0), "r"(c4) : "memory");
}

template <int S, int TAIL, int NXT, int NYT, int PF>
struct B3Cfg {
    static constexpr int T = TAIL ? 1 : 0;
    static constexpr int HX = 4, H = 4;                  // halo in x and y: even, so tiles start on an x-pair and a row pair
    static constexpr int ZH = S + T;                     // halo in z (planes before / after the segment)
    static constexpr int TX = NXT - 2 * HX, TY = NYT - 2 * H;
    static constexpr int NXP = NXT / 2, NPH = NXP * (NYT / 2);   // x-pairs per row, 2x2 patches per plane (= live threads)
    static constexpr int NT = (NPH + 31) / 32 * 32;
    static constexpr int R = (S + T + 3) / 2 * 2;        // register rings: planes zl .. zl-S-1-T, period even
    static constexpr int NS = S + T + 1 + PF;            // TMA ring (phi, wx, wy): planes zl+PF .. zl-S-T
    static constexpr int NP = S + T;                     // private ring (rhs, 1/D): planes zl-1 .. zl-S-T
    static constexpr int ARR = 4 * NPH;                  // one array of one plane: [x-parity][row parity][NPH]
    static constexpr int TSLOT = 3 * ARR, PSLOT = 2 * ARR;
    static constexpr size_t SMEM_DATA = (size_t)(NS * TSLOT + NP * PSLOT) * sizeof(double);
    static constexpr size_t SMEM = SMEM_DATA + (NS + 1) * sizeof(uint64_t) + 128;   // + mbarriers, + alignment slack
    static constexpr uint32_t TX_BYTES = (uint32_t)(TSLOT * sizeof(double));
    static_assert(S >= 1 && S + T <= 4 && TX > 0 && TY > 0 && NXT % 4 == 0 && NYT % 2 == 0 && NPH % 4 == 0 &&
                      R >= S + 2 + T && R % 2 == 0 && PF >= 1, "tile");
};

template <int S, int TAIL, bool PROLONG, int C0, int NXT, int NYT, int PF>
__global__ void __launch_bounds__(B3Cfg<S, TAIL, NXT, NYT, PF>::NT, 1) smooth_block3_kernel(const __grid_constant__ Block3Args g)
{
    using C = B3Cfg<S, TAIL, NXT, NYT, PF>;
    constexpr int NXP = C::NXP, NPH = C::NPH, R = C::R, NS = C::NS, NP = C::NP, ARR = C::ARR;
    constexpr int TSLOT = C::TSLOT, PSLOT = C::PSLOT;
    constexpr int A_PHI = 0, A_WX = ARR, A_WY = 2 * ARR, B_RHS = 0, B_DINV = ARR;
    constexpr int XB = 2 * NPH;                     // offset of the odd-x block inside an array
    extern __shared__ __align__(128) double b3_smem[];   // (indexed as an array: the accesses must stay LDS / STS, not generic loads)
    double* const ring = b3_smem;
    double* const priv = ring + NS * TSLOT;
    uint64_t* const full = reinterpret_cast<uint64_t*>(priv + NP * PSLOT);
    uint64_t* const stepbar = full + NS;

    const bool live = threadIdx.x < NPH;
    const int t = live ? threadIdx.x : 0;          // idle lanes of the last warp shadow thread 0 (and commit nothing)
    const int m = t % NXP, jj = t / NXP;
    const int lane = threadIdx.x & 31;

    // planes before the first loaded one: zero weights and zero 1/D keep them at zero (finite)
    for (int q = threadIdx.x; q < NS * TSLOT + NP * PSLOT; q += C::NT) ring[q] = 0.0;
    if (threadIdx.x == 0) {
        for (int k = 0; k < NS; ++k) mbar_init(full + k, 1);
        mbar_init(stepbar, C::NT / 32);
        fence_mbar_init();
    }
    fence_proxy_async();                           // the zeros (generic proxy) before the TMA writes (async proxy)
    __syncthreads();

    // CTA -> (tile, z-segment), tile index fastest; segments are cut at even z (restriction pairs stay together)
    const int ntiles = g.ntx * g.nty;
    const int tile = (int)(blockIdx.x % ntiles), seg = (int)(blockIdx.x / ntiles);
    const int za = (int)((long long)(g.G.nz / 2) * seg / g.nzseg) * 2;
    const int zb = seg == g.nzseg - 1 ? g.G.nz : (int)((long long)(g.G.nz / 2) * (seg + 1) / g.nzseg) * 2;
    const int tx = tile % g.ntx, ty = tile / g.ntx;
    const int m0 = (tx * C::TX - C::HX) / 2, jj0 = (ty * C::TY - C::H) / 2;   // box origin: x-pair, row pair
    const int gx = 2 * (m0 + m), gy0 = 2 * (jj0 + jj);                        // rows gy0 and gy0 + 1
    const bool in_x = live && gx >= 0 && gx < g.G.nx;
    const bool in_p = in_x && gy0 >= 0 && gy0 < g.G.ny;                       // ny is even: both rows or none
    const bool int_x = m >= C::HX / 2 && m < C::HX / 2 + C::TX / 2;
    const bool interior = in_p && int_x && 2 * jj >= C::H && 2 * jj < C::H + C::TY;
    // rows 0 and NYT-1 and the first / last column of the tile are rim: never relaxed.  ok[r][sg]: row r, x-parity sg
    const bool ok[2][2] = {{live && jj >= 1 && m > 0, live && jj >= 1 && m < NXP - 1},
                           {live && jj <= NYT / 2 - 2 && m > 0, live && jj <= NYT / 2 - 2 && m < NXP - 1}};
    // the x-pair's even cell in row gy0 of plane 0 (internal layout); its odd cell is `odd` further on
    const long long cbase = (long long)g.G.pitch * gy0 + (gx >> 1);
    const int odd = g.G.hp;

    // register rings [row][slot]: even-x / odd-x phi and wz of this thread's pair; iteration n lives in slot n % R
    double pe[2][R], po[2][R], we[2][R], wo[2][R];
#pragma unroll
    for (int r = 0; r < 2; ++r)
#pragma unroll
        for (int k = 0; k < R; ++k) pe[r][k] = po[r][k] = we[r][k] = wo[r][k] = 0.0;

    // private loads in flight: wz (and the coarse correction) of the next plane; rhs, 1/D of the current one
    double2 r_wz[2], r_rhs[2], r_dinv[2];
    double r_e = 0.0;
    auto ld2 = [&](const double* p, long long c) { return make_double2(__ldg(p + c), __ldg(p + c + odd)); };
    auto issue_wz = [&](int zq) {
        const bool z_in = in_p && zq >= 0 && zq < g.G.nz;
        r_e = 0.0;
#pragma unroll
        for (int r = 0; r < 2; ++r) {
            r_wz[r] = make_double2(0.0, 0.0);
            if (z_in) r_wz[r] = ld2(g.wz, cbase + r * g.G.pitch + g.G.plane * zq);
        }
        if (PROLONG && z_in) r_e = __ldg(g.e + cell_at(g.CG, gx >> 1, gy0 >> 1, zq >> 1));
    };
    auto issue_rd = [&](int zq) {
        const bool z_in = in_p && zq >= 0 && zq < g.G.nz;
#pragma unroll
        for (int r = 0; r < 2; ++r) {
            r_rhs[r] = r_dinv[r] = make_double2(0.0, 0.0);
            if (z_in) {
                const long long c = cbase + r * g.G.pitch + g.G.plane * zq;
                r_rhs[r] = ld2(g.rhs, c);
                r_dinv[r] = ld2(g.dinv, c);
            }
        }
    };
    auto tma_plane = [&](int slot, int z) {        // one elected thread
        double* dst = ring + slot * TSLOT;
        mbar_expect_tx(full + slot, C::TX_BYTES);
        tma_load_5d(dst + A_PHI, &g.tm_phi, full + slot, m0, jj0, z);
        tma_load_5d(dst + A_WX, &g.tm_wx, full + slot, m0, jj0, z);
        tma_load_5d(dst + A_WY, &g.tm_wy, full + slot, m0, jj0, z);
    };

    const int z0 = za - C::ZH;
    const int niter = (zb - za) + 2 * C::ZH;       // iteration n: zl = z0 + n; the last final plane zb-1 = zl - S (- T for the tail)
    if (threadIdx.x == 0) {
#pragma unroll
        for (int q = 0; q < PF; ++q)
            if (q < niter) tma_plane(q, z0 + q);
    }
    issue_wz(z0);

    double nrm = 0.0;
    bool nrm_nan = false;
    double acc = 0.0;    // BT_RESTRICT: running sum over the children of one coarse cell (even plane, then odd plane)
    int slotn = 0, phasen = 0, pn = 0;             // n % NS, (n / NS) & 1, n % NP

    for (int nbase = 0; nbase < niter; nbase += R) {
#pragma unroll
        for (int u = 0; u < R; ++u) {
            const int n = nbase + u;               // n % R == u (compile time: ring indices, parities)
            if (n >= niter) break;                 // uniform
            const int zl = z0 + n;

            // ---- A: plane zl has landed: its own columns enter the register rings ----
            mbar_wait(full + slotn, (uint32_t)phasen);
            {
                double* P0 = ring + slotn * TSLOT + t;
#pragma unroll
                for (int r = 0; r < 2; ++r) {
                    double a = P0[A_PHI + r * NPH], b = P0[A_PHI + XB + r * NPH];
                    if (PROLONG) {                 // S4: phi += P e while loading; the neighbours read the corrected plane
                        a += r_e; b += r_e;
                        if (live) { P0[A_PHI + r * NPH] = a; P0[A_PHI + XB + r * NPH] = b; }
                    }
                    pe[r][u] = a; po[r][u] = b;
                    we[r][u] = r_wz[r].x; wo[r][u] = r_wz[r].y;
                }
            }
            issue_wz(zl + 1);
            issue_rd(zl);

            // ---- B: every thread has finished iteration n-1 ----
            if (n > 0) mbar_wait(stepbar, (uint32_t)((n - 1) & 1));
            if (threadIdx.x == 0) {
                if (n + PF < niter) {
                    int sl = slotn + PF; if (sl >= NS) sl -= NS;
                    tma_plane(sl, zl + PF);
                }
                if (n + PF + 2 < niter && zl + PF + 2 < g.G.nz) {
                    tma_prefetch_5d(&g.tm_phi, m0, jj0, zl + PF + 2);
                    tma_prefetch_5d(&g.tm_wx, m0, jj0, zl + PF + 2);
                    tma_prefetch_5d(&g.tm_wy, m0, jj0, zl + PF + 2);
                }
            }

            // ---- C: stages: half-sweep s on plane zl - s (register slot (u-s) % R); rim threads compute and discard.
            // Row r relaxes its cell of x-parity sg = (C0 + r + zl + 1) & 1 = (C0 + r + u + 1 + ZH) & 1 (za, gy0 and gx are even). ----
#pragma unroll
            for (int s = 1; s <= S; ++s) {
                const int c = ((u - s) % R + R) % R, cu = ((u - s + 1) % R + R) % R, cd = ((u - s - 1) % R + R) % R;
                int sl = slotn - s; if (sl < 0) sl += NS;
                int ps = pn - s; if (ps < 0) ps += NP;
                double* P = ring + sl * TSLOT + t;
                const double* Q = priv + ps * PSLOT + t;
                double nv[2];
#pragma unroll
                for (int r = 0; r < 2; ++r) {
                    const int sg = (C0 + r + u + 1 + C::ZH) & 1;
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
                    nv[r] = Q[B_DINV + oA] * (Q[B_RHS + oA] + v);
                }
#pragma unroll
                for (int r = 0; r < 2; ++r) {
                    const int sg = (C0 + r + u + 1 + C::ZH) & 1;
                    if (ok[r][sg]) {
                        if (sg) po[r][c] = nv[r]; else pe[r][c] = nv[r];
                        P[A_PHI + sg * XB + r * NPH] = nv[r];
                    }
                }
            }

            // ---- residual stage on plane zl - S - 1; all its neighbours are final: plane zl - S in this thread's
            // registers (just relaxed), the others since the previous iteration ----
            if (TAIL != BT_NONE) {
                const int pr = zl - S - 1;
                if (pr >= za && pr < zb && interior) {
                    const int k = ((u - S - 1) % R + R) % R, ku = ((u - S) % R + R) % R, kd = ((u - S - 2) % R + R) % R;
                    int sl = slotn - (S + 1); if (sl < 0) sl += NS;
                    int ps = pn - (S + 1); if (ps < 0) ps += NP;
                    const double* P = ring + sl * TSLOT + t;
                    const double* Q = priv + ps * PSLOT + t;
                    double res[2][2];                    // [row][x-parity]
#pragma unroll
                    for (int r = 0; r < 2; ++r)
#pragma unroll
                        for (int e = 0; e < 2; ++e) {
                            const int o = e * XB + r * NPH;
                            const double ce = e ? po[r][k] : pe[r][k], mate = e ? pe[r][k] : po[r][k];
                            const double xo = P[A_PHI + (e ? r * NPH + 1 : XB + r * NPH - 1)];
                            const double yo = P[A_PHI + e * XB + (r ? NXP : NPH - NXP)];
                            const double yin = e ? po[1 - r][k] : pe[1 - r][k];
                            const double xm = e ? mate : xo, xp = e ? xo : mate;
                            const double ym = r ? yin : yo, yp = r ? yo : yin;
                            double v = P[A_WX + o] * xm;
                            v = fma(P[A_WX + (e ? r * NPH + 1 : XB + r * NPH)], xp, v);
                            v = fma(P[A_WY + o], ym, v);
                            v = fma(P[A_WY + e * XB + (r ? NXP : NPH)], yp, v);
                            v = fma(e ? wo[r][k] : we[r][k], e ? po[r][kd] : pe[r][kd], v);
                            v = fma(e ? wo[r][ku] : we[r][ku], e ? po[r][ku] : pe[r][ku], v);
                            res[r][e] = Q[B_RHS + o] + v - ce / Q[B_DINV + o];
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

            // ---- D: this thread's shared-memory writes of iteration n are done ----
            fence_proxy_async();                   // they precede the TMA write that will reuse the slot
            __syncwarp();
            if (lane == 0) mbar_arrive(stepbar);

            // ---- E: plane zl - S is final: write it back from registers ----
            {
                const int p = zl - S, c = ((u - S) % R + R) % R;
                if (p >= za && p < zb && interior) {
#pragma unroll
                    for (int r = 0; r < 2; ++r) {
                        double* q = g.phi_out + cbase + r * g.G.pitch + g.G.plane * p;
                        q[0] = pe[r][c]; q[odd] = po[r][c];
                    }
                }
            }
            // ---- F: rhs and 1/D of plane zl take the private slot that plane zl - S - T just vacated ----
            if (live) {
                double* F = priv + pn * PSLOT + t;
#pragma unroll
                for (int r = 0; r < 2; ++r) {
                    F[B_RHS + r * NPH] = r_rhs[r].x;   F[B_RHS + XB + r * NPH] = r_rhs[r].y;
                    F[B_DINV + r * NPH] = r_dinv[r].x; F[B_DINV + XB + r * NPH] = r_dinv[r].y;
                }
            }
            if (++slotn == NS) { slotn = 0; phasen ^= 1; }
            if (++pn == NP) pn = 0;
        }
    }

    if (TAIL == BT_NORM) {
        if (nrm_nan) nrm = __longlong_as_double(0x7ff8000000000000ll);
        block_max_to_global(nrm, g.norm_out);
    }
}


// ------------------------------------------------------------------------------------------------
// Row variant: one thread per x-pair of ONE row (twice the threads of the 2 x 2 patch variant, half the registers each:
// the ncu capture of the patch variant shows 11 warps per SM waiting on their own LDS -> DFMA chains, nothing saturated).
// 9 LDS.64 + 1 STS.64 per relaxation instead of 8 + 1 (both y-neighbours come from shared memory).  The array is the 4-D
// tensor (m, row, x-parity, plane), a box {NXP, NYT, 2, 1} lands as [x-parity][row][m]; the y halo is S + T rows, not
// rounded up to even.  A thread calls its two cells by when they are relaxed, not by x-parity: cell L (0 / 1) is the one
// relaxed in iterations of parity L, so every register index stays a compile-time constant although rows of both parities
// share a warp; what depends on the row's parity are three shared-memory offsets per cell, computed once.
// BT_RESTRICT: the two rows of a coarse cell belong to two threads; the odd row's x-pair sum goes through a small
// shared-memory scratch and is consumed by the even row's thread one iteration later (after the step barrier), in the
// order residual_restrict_kernel sums the children.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void tma_load_4d(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1, int c3)
{
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(0), "r"(c3) : "memory");
}
__device__ __forceinline__ void tma_prefetch_4d(const CUtensorMap* map, int c0, int c1, int c3)
{
    asm volatile("cp.async.bulk.prefetch.tensor.4d.L2.global [%0, {%1, %2, %3, %4}];"
                 ::"l"(map), "r"(c0), "r"(c1), "r"(0), "r"(c3) : "memory");
}

template <int S, int TAIL, int NXT, int NYT, int PF>
struct B3rCfg {
    static constexpr int T = TAIL ? 1 : 0;
    static constexpr int H = S + T;                      // halo in y
    static constexpr int HX = H <= 4 ? 4 : (H + 1) / 2 * 2;   // halo in x: even (tiles start on an x-pair), >= 4 (32-byte aligned)
    static constexpr int ZH = S + T;
    static constexpr int TX = NXT - 2 * HX, TY = NYT - 2 * H;
    static constexpr int NXP = NXT / 2, NPH = NXP * NYT; // x-pairs per row, x-pairs per plane (= live threads)
    static constexpr int NT = (NPH + 31) / 32 * 32;
    static constexpr int R = (S + T + 3) / 2 * 2;
    static constexpr int NS = S + T + 1 + PF, NP = S + T;
    static constexpr int ARR = 2 * NPH;                  // one array of one plane: [x-parity][NPH]
    static constexpr int TSLOT = 3 * ARR, PSLOT = 2 * ARR;
    static constexpr int SCRATCH = TAIL == BT_RESTRICT ? 2 * NPH : 0;
    static constexpr size_t SMEM_DATA = (size_t)(NS * TSLOT + NP * PSLOT + SCRATCH) * sizeof(double);
    static constexpr size_t SMEM = SMEM_DATA + 256;      // + front pad (mbarriers)
    static constexpr uint32_t TX_BYTES = (uint32_t)(TSLOT * sizeof(double));
    static_assert(S >= 1 && S + T <= 7 && TX > 0 && TY > 0 && TY % 2 == 0 && NXT % 4 == 0 && (ARR * 8) % 128 == 0 &&
                      R >= S + 2 + T && R % 2 == 0 && PF >= 1, "tile");
};

template <int S, int TAIL, bool PROLONG, int C0, int NXT, int NYT, int PF>
__global__ void __launch_bounds__(B3rCfg<S, TAIL, NXT, NYT, PF>::NT, 1) smooth_block3r_kernel(const __grid_constant__ Block3Args g)
{
    using C = B3rCfg<S, TAIL, NXT, NYT, PF>;
    constexpr int NXP = C::NXP, NPH = C::NPH, R = C::R, NS = C::NS, NP = C::NP, ARR = C::ARR;
    constexpr int TSLOT = C::TSLOT, PSLOT = C::PSLOT;
    constexpr int A_PHI = 0, A_WX = ARR, A_WY = 2 * ARR, B_RHS = 0, B_DINV = ARR;
    constexpr int XB = NPH;                         // offset of the odd-x block inside an array
    extern __shared__ __align__(128) double b3_smem[];
    // the first 256 bytes hold the mbarriers and keep the y-neighbour reads of the first row (rim: computed and
    // discarded) inside the allocation
    double* const ring = b3_smem + 32;
    double* const priv = ring + NS * TSLOT;
    double* const scratch = priv + NP * PSLOT;
    uint64_t* const full = reinterpret_cast<uint64_t*>(b3_smem);
    uint64_t* const stepbar = full + NS;
    static_assert((NS + 1) * 8 + NXP * 8 <= 256, "front pad");

    const bool live = threadIdx.x < NPH;
    const int t = live ? threadIdx.x : 0;
    const int m = t % NXP, j = t / NXP;
    const int lane = threadIdx.x & 31;

    for (int q = threadIdx.x; q < NS * TSLOT + NP * PSLOT + C::SCRATCH; q += C::NT) ring[q] = 0.0;
    if (threadIdx.x == 0) {
        for (int k = 0; k < NS; ++k) mbar_init(full + k, 1);
        mbar_init(stepbar, C::NT / 32);
        fence_mbar_init();
    }
    fence_proxy_async();
    __syncthreads();

    const int ntiles = g.ntx * g.nty;
    const int tile = (int)(blockIdx.x % ntiles), seg = (int)(blockIdx.x / ntiles);
    const int za = (int)((long long)(g.G.nz / 2) * seg / g.nzseg) * 2;
    const int zb = seg == g.nzseg - 1 ? g.G.nz : (int)((long long)(g.G.nz / 2) * (seg + 1) / g.nzseg) * 2;
    const int tx = tile % g.ntx, ty = tile / g.ntx;
    const int m0 = (tx * C::TX - C::HX) / 2, j0 = ty * C::TY - C::H;          // box origin: x-pair, row
    const int gx = 2 * (m0 + m), gy = j0 + j;
    const bool in_p = live && gx >= 0 && gx < g.G.nx && gy >= 0 && gy < g.G.ny;
    const bool interior = in_p && m >= C::HX / 2 && m < C::HX / 2 + C::TX / 2 && j >= C::H && j < C::H + C::TY;
    // cell L of this thread is relaxed in iterations n with n % 2 == L: its x-parity p0 ^ L, where
    // p0 = (C0 + 1 + ZH + gy) & 1 (cell (x, y, z) has colour (x + y + z) & 1; stage s in iteration n relaxes colour
    // C0 + s - 1 on plane z0 + n - s; za and gx are even)
    const int p0 = (C0 + 1 + C::ZH + gy) & 1;
    int oA[2], oX[2], oW[2];                        // per cell: itself, its x-neighbour outside the pair, its high-x weight
    bool ok[2];                                     // rim cells (first / last row, first / last cell of a row) are never relaxed
#pragma unroll
    for (int L = 0; L < 2; ++L) {
        const int sg = p0 ^ L;
        oA[L] = sg * XB + t;
        oX[L] = sg ? t + 1 : XB + t - 1;
        oW[L] = sg ? t + 1 : XB + t;
        ok[L] = live && j >= 1 && j <= NYT - 2 && (sg ? m < NXP - 1 : m > 0);
    }
    const long long cbase = (long long)g.G.pitch * gy + (gx >> 1);
    const int odd = g.G.hp;

    // register rings [cell L][slot]: phi and wz of this thread's pair; iteration n lives in slot n % R
    double ph[2][R], wz[2][R];
#pragma unroll
    for (int L = 0; L < 2; ++L)
#pragma unroll
        for (int k = 0; k < R; ++k) ph[L][k] = wz[L][k] = 0.0;

    double r_wz[2], r_rhs[2], r_dinv[2];            // [x-parity]
    double r_e = 0.0;
    auto issue_wz = [&](int zq) {
        const bool z_in = in_p && zq >= 0 && zq < g.G.nz;
        r_wz[0] = r_wz[1] = 0.0; r_e = 0.0;
        if (z_in) {
            const long long c = cbase + g.G.plane * zq;
            r_wz[0] = __ldg(g.wz + c); r_wz[1] = __ldg(g.wz + c + odd);
            if (PROLONG) r_e = __ldg(g.e + cell_at(g.CG, gx >> 1, gy >> 1, zq >> 1));
        }
    };
    auto issue_rd = [&](int zq) {
        const bool z_in = in_p && zq >= 0 && zq < g.G.nz;
        r_rhs[0] = r_rhs[1] = r_dinv[0] = r_dinv[1] = 0.0;
        if (z_in) {
            const long long c = cbase + g.G.plane * zq;
            r_rhs[0] = __ldg(g.rhs + c); r_rhs[1] = __ldg(g.rhs + c + odd);
            r_dinv[0] = __ldg(g.dinv + c); r_dinv[1] = __ldg(g.dinv + c + odd);
        }
    };
    auto tma_plane = [&](int slot, int z) {
        double* dst = ring + slot * TSLOT;
        mbar_expect_tx(full + slot, C::TX_BYTES);
        tma_load_4d(dst + A_PHI, &g.tm_phi, full + slot, m0, j0, z);
        tma_load_4d(dst + A_WX, &g.tm_wx, full + slot, m0, j0, z);
        tma_load_4d(dst + A_WY, &g.tm_wy, full + slot, m0, j0, z);
    };

    const int z0 = za - C::ZH;
    const int niter = (zb - za) + 2 * C::ZH;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int q = 0; q < PF; ++q)
            if (q < niter) tma_plane(q, z0 + q);
    }
    issue_wz(z0);

    double nrm = 0.0;
    bool nrm_nan = false;
    double acc = 0.0, rsum_prev = 0.0;             // BT_RESTRICT (even rows): running sum of a coarse cell, this row's last x-pair sum
    int slotn = 0, phasen = 0, pn = 0;

    // BT_RESTRICT: the children of plane pr (tail of the previous iteration): even row (this thread), then odd row (scratch)
    auto consume_restrict = [&](int pr, int par) {
        if (pr >= za && pr < zb && interior && !(gy & 1)) {
            acc += rsum_prev;
            acc += scratch[par * NPH + t + NXP];
            if (pr & 1) {
                const long long cc = cell_at(g.CG, gx >> 1, gy >> 1, pr >> 1);
                g.crhs[cc] = acc / 8.0;
                g.cphi[cc] = 0.0;
                acc = 0.0;
            }
        }
    };

    for (int nbase = 0; nbase < niter; nbase += R) {
#pragma unroll
        for (int u = 0; u < R; ++u) {
            const int n = nbase + u;
            if (n >= niter) break;
            const int zl = z0 + n;

            // ---- A: plane zl has landed: its own cells enter the register rings ----
            mbar_wait(full + slotn, (uint32_t)phasen);
            {
                double* P0 = ring + slotn * TSLOT;
#pragma unroll
                for (int L = 0; L < 2; ++L) {
                    double a = P0[A_PHI + oA[L]];
                    if (PROLONG) { a += r_e; if (live) P0[A_PHI + oA[L]] = a; }
                    ph[L][u] = a;
                    wz[L][u] = (p0 ^ L) ? r_wz[1] : r_wz[0];
                }
            }
            issue_wz(zl + 1);
            issue_rd(zl);

            // ---- B: every thread has finished iteration n-1 ----
            if (n > 0) mbar_wait(stepbar, (uint32_t)((n - 1) & 1));
            if (threadIdx.x == 0) {
                if (n + PF < niter) {
                    int sl = slotn + PF; if (sl >= NS) sl -= NS;
                    tma_plane(sl, zl + PF);
                }
                if (n + PF + 2 < niter && zl + PF + 2 < g.G.nz) {
                    tma_prefetch_4d(&g.tm_phi, m0, j0, zl + PF + 2);
                    tma_prefetch_4d(&g.tm_wx, m0, j0, zl + PF + 2);
                    tma_prefetch_4d(&g.tm_wy, m0, j0, zl + PF + 2);
                }
            }
            if (TAIL == BT_RESTRICT) consume_restrict(zl - 1 - S - 1, (n - 1) & 1);

            // ---- C: stage s relaxes cell L = u & 1 of plane zl - s (register slot (u-s) % R) ----
            const int L = u & 1;
#pragma unroll
            for (int s = 1; s <= S; ++s) {
                const int c = ((u - s) % R + R) % R, cu = ((u - s + 1) % R + R) % R, cd = ((u - s - 1) % R + R) % R;
                int sl = slotn - s; if (sl < 0) sl += NS;
                int ps = pn - s; if (ps < 0) ps += NP;
                double* P = ring + sl * TSLOT;
                const double* Q = priv + ps * PSLOT;
                const double mate = ph[1 - L][c], xo = P[A_PHI + oX[L]];
                const bool sg = (p0 ^ L) != 0;
                const double xm = sg ? mate : xo, xp = sg ? xo : mate;
                double v = P[A_WX + oA[L]] * xm;
                v = fma(P[A_WX + oW[L]], xp, v);
                v = fma(P[A_WY + oA[L]], P[A_PHI + oA[L] - NXP], v);
                v = fma(P[A_WY + oA[L] + NXP], P[A_PHI + oA[L] + NXP], v);
                v = fma(wz[L][c], ph[L][cd], v);
                v = fma(wz[L][cu], ph[L][cu], v);
                const double nv = Q[B_DINV + oA[L]] * (Q[B_RHS + oA[L]] + v);
                if (ok[L]) { ph[L][c] = nv; P[A_PHI + oA[L]] = nv; }
            }

            // ---- residual stage on plane zl - S - 1 (all its neighbours are final) ----
            if (TAIL != BT_NONE) {
                const int pr = zl - S - 1;
                if (pr >= za && pr < zb && interior) {
                    const int k = ((u - S - 1) % R + R) % R, ku = ((u - S) % R + R) % R, kd = ((u - S - 2) % R + R) % R;
                    int sl = slotn - (S + 1); if (sl < 0) sl += NS;
                    int ps = pn - (S + 1); if (ps < 0) ps += NP;
                    const double* P = ring + sl * TSLOT;
                    const double* Q = priv + ps * PSLOT;
                    double res[2];                       // [cell L]
#pragma unroll
                    for (int LL = 0; LL < 2; ++LL) {
                        const double ce = ph[LL][k], mate = ph[1 - LL][k], xo = P[A_PHI + oX[LL]];
                        const bool sg = (p0 ^ LL) != 0;
                        const double xm = sg ? mate : xo, xp = sg ? xo : mate;
                        double v = P[A_WX + oA[LL]] * xm;
                        v = fma(P[A_WX + oW[LL]], xp, v);
                        v = fma(P[A_WY + oA[LL]], P[A_PHI + oA[LL] - NXP], v);
                        v = fma(P[A_WY + oA[LL] + NXP], P[A_PHI + oA[LL] + NXP], v);
                        v = fma(wz[LL][k], ph[LL][kd], v);
                        v = fma(wz[LL][ku], ph[LL][ku], v);
                        res[LL] = Q[B_RHS + oA[LL]] + v - ce / Q[B_DINV + oA[LL]];
                    }
                    if (TAIL == BT_NORM) {
#pragma unroll
                        for (int LL = 0; LL < 2; ++LL) {
                            const double a = fabs(res[LL]);
                            nrm_nan |= (a != a);
                            nrm = fmax(nrm, a);
                        }
                    }
                    if (TAIL == BT_RESTRICT) {
                        const double rs = p0 ? res[1] + res[0] : res[0] + res[1];   // even-x child first
                        if (gy & 1) scratch[(n & 1) * NPH + t] = rs; else rsum_prev = rs;
                    }
                }
            }

            // ---- D: this thread's shared-memory writes of iteration n are done ----
            fence_proxy_async();
            __syncwarp();
            if (lane == 0) mbar_arrive(stepbar);

            // ---- E: plane zl - S is final: write it back from registers ----
            {
                const int p = zl - S, c = ((u - S) % R + R) % R;
                if (p >= za && p < zb && interior) {
                    double* q = g.phi_out + cbase + g.G.plane * p;
                    q[0] = p0 ? ph[1][c] : ph[0][c];
                    q[odd] = p0 ? ph[0][c] : ph[1][c];
                }
            }
            // ---- F: rhs and 1/D of plane zl take the private slot that plane zl - S - T just vacated ----
            if (live) {
                double* F = priv + pn * PSLOT + t;
                F[B_RHS] = r_rhs[0];   F[B_RHS + XB] = r_rhs[1];
                F[B_DINV] = r_dinv[0]; F[B_DINV + XB] = r_dinv[1];
            }
            if (++slotn == NS) { slotn = 0; phasen ^= 1; }
            if (++pn == NP) pn = 0;
        }
    }

    if (TAIL == BT_RESTRICT) {                       // the last plane's children
        mbar_wait(stepbar, (uint32_t)((niter - 1) & 1));
        consume_restrict(z0 + niter - 1 - S - 1, (niter - 1) & 1);
    }
    if (TAIL == BT_NORM) {
        if (nrm_nan) nrm = __longlong_as_double(0x7ff8000000000000ll);
        block_max_to_global(nrm, g.norm_out);
    }
}

}  // namespace vmg
