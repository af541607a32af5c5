// vmg_sched.cuh -- sequencing of one V-cycle (S7): which kernel runs each step on each level, plain
// launches or one CUDA graph replay (north_star (4)).
//   levels 0 .. tail_level-1 : one launch per colour half-sweep / transfer, in an order that reuses L2 (next_dir), with
//                              programmatic dependent launch; with option blocked = 1 the blocked passes of
//                              vmg_block2.cuh where the level qualifies
//   levels tail_level .. last: one single-CTA launch (vmg_tail.cuh)
#pragma once
#include "vmg_internal.h"
#include "vmg_kernels.cuh"
#include "vmg_tail.cuh"
#include "vmg_cluster.cuh"
#include "vmg_block2.cuh"
#include "vmg_block3.cuh"
#include "../../include/vmg.h"
#include <algorithm>
#include <cstring>
#include <mutex>

namespace vmg {

inline LevelView view(const VmgLevel& L)
{
    LevelView v;
    v.wx = L.wx; v.wy = L.wy; v.wz = L.wz; v.dinv = L.dinv;
    v.G = L.G;
    v.cx = L.cx; v.cy = L.cy; v.cz = L.cz; v.cw = L.cw; v.mk = L.mk;
    v.pstride = L.pstride; v.nprob = L.nprob;
    return v;
}

// picks the instantiation for the level's kind of weights (LevelView::cw)
#define VMG_BY_WEIGHTS(L, KERNEL) ((L).cw == 2 ? KERNEL<2> : (L).cw ? KERNEL<1> : KERNEL<0>)

inline unsigned grid_for(long long n) { return (unsigned)cdiv(n, kThreads); }
inline unsigned conv_grid(long long n) { return (unsigned)cdiv(cdiv(n, kConvElems), kThreads); }   // fold_bc, to_internal, to_natural: kConvElems elements per thread

// launch shape of the kernels that take one x-pair slot per thread: block (x-pairs, rows) of kThreads threads with as many
// x-pairs as the row has (whole warps, at most 128), grid (x-pair blocks, row blocks, planes)
inline void cell_launch_dims(const Geom& G, dim3& grid, dim3& block)
{
    const int bx = std::min(128, 32 * ((G.nx + 31) / 32)), by = kThreads / bx;
    block = dim3(bx, by, 1);
    grid = dim3((G.nx + bx - 1) / bx, (G.ny + by - 1) / by, G.nz);
}

inline void pair_launch_dims(const VmgLevel& L, dim3& grid, dim3& block)
{
    const int bx = std::min(128, 32 * ((L.G.ne + 31) / 32)), by = kThreads / bx;
    block = dim3(bx, by, 1);
    grid = dim3((L.G.ne + bx - 1) / bx, (L.ny + by - 1) / by, L.nz * L.nprob);   // batched capture: planes x problems
}

// direction of the next whole-level kernel: consecutive kernels walk the level in opposite directions (L2 reuse)
inline int next_dir(vmg_s* h, VmgLevel& L) { int d = h->snake ? L.dir : 0; L.dir ^= 1; return d; }

// launch with programmatic stream serialisation (see grid_dependency_wait in vmg_kernels.cuh)
template <typename... KArgs, typename... Args>
inline void launch_pdl(vmg_s* h, void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, Args... args)
{
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = h->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = h->use_pdl ? 1 : 0;
    cfg.attrs = at; cfg.numAttrs = 1;
    cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

inline double* cur_phi(VmgLevel& L) { return L.cur ? L.phi2 : L.phi; }
inline double* other_phi(VmgLevel& L) { return L.cur ? L.phi : L.phi2; }

// RAII event pair around a group of launches of one kernel class (only when option "profile" is on).
struct ProfScope {
    vmg_s* h; int cls; long long* counter; long long before; cudaEvent_t start = nullptr;
    ProfScope(vmg_s* h_, int cls_, long long* counter_) : h(h_), cls(cls_), counter(counter_), before(counter_ ? *counter_ : 0)
    {
        if (!h->profile) return;
        start = take();
        cudaEventRecord(start, h->stream);
    }
    ~ProfScope()
    {
        if (!h->profile) return;
        cudaEvent_t stop = take();
        cudaEventRecord(stop, h->stream);
        h->prof_pending.push_back({cls, counter ? *counter - before : 1, start, stop});
    }
    cudaEvent_t take()
    {
        cudaEvent_t e;
        if (!h->prof_pool.empty()) { e = h->prof_pool.back(); h->prof_pool.pop_back(); }
        else cudaEventCreate(&e);
        return e;
    }
};

// after a stream synchronise: fold the pending event pairs into the per-class totals
inline void prof_collect(vmg_s* h)
{
    for (auto& p : h->prof_pending) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, p.start, p.stop) == cudaSuccess) {
            h->prof_ms[p.cls] += ms;
            h->prof_launches[p.cls] += p.launches;
        }
        h->prof_pool.push_back(p.start);
        h->prof_pool.push_back(p.stop);
    }
    h->prof_pending.clear();
    (void)cudaGetLastError();
}

// bt: the level-0 internal array, or (bt_natural) a caller array in the public layout
inline int enqueue_fold_bc(vmg_s* h, const double* rhs, double* bt, bool bt_natural = false, unsigned long long* norm_out = nullptr)
{
    VmgLevel& L = h->lev[0];
    FoldArgs g;
    g.norm_out = norm_out;
    g.rhs = rhs; g.bt = bt;
    for (int f = 0; f < 6; ++f) {
        g.wb[f] = L.wb[f];
        g.val[f] = h->bc_has_value[f] ? h->bcval[f] : nullptr;
        g.dirichlet[f] = h->bctype[f] == VMG_BC_DIRICHLET;
    }
    g.G = L.G; g.three_d = h->three_d; g.bt_natural = bt_natural;
    g.mask = h->d_mask; g.mfold = h->m_fold;
    g.h[0] = L.hx; g.h[1] = L.hy; g.h[2] = L.hz;
    {
        ProfScope ps(h, VMG_PC_FOLD, nullptr);
        fold_bc_kernel<<<conv_grid(L.n), kThreads, 0, h->stream>>>(g);
    }
    h->launches += 1;
    return cudaGetLastError() == cudaSuccess ? VMG_OK : VMG_ERR_CUDA;
}

// ------------------------------------------------------------------------------------------------
// plain path: one launch per step, in place on the level's current phi buffer
// ------------------------------------------------------------------------------------------------
// skip_first: number of leading half-sweeps already done by the caller
// first: colour of the first half-sweep of every sweep (1: black -> red, the adjoint order of the symmetric V-cycle)
inline void plain_smooth(vmg_s* h, int l, int nsweeps, long long* count, int skip_first = 0, int first = 0)
{
    VmgLevel& L = h->lev[l];
    LevelView v = view(L);
    for (int s = 0; s < nsweeps; ++s)
        for (int c2 = 0; c2 < 2; ++c2) {
            const int colour = (first + c2) & 1;
            if (2 * s + c2 < skip_first) continue;
            dim3 grid, block;
            pair_launch_dims(L, grid, block);
            if (L.cw == 0 && L.n >= h->phi_keep_cells)
                launch_pdl(h, smooth_colour_kernel<0, 1>, grid, block, 0, v, cur_phi(L), L.rhs, colour, next_dir(h, L));
            else
                launch_pdl(h, VMG_BY_WEIGHTS(L, smooth_colour_kernel), grid, block, 0, v, cur_phi(L), L.rhs, colour, next_dir(h, L));
            ++*count;
        }
}

// after_black: the level's last kernel was a black half-sweep (pre-smoothing with nu1 >= 1): on levels of at least
// restrict_red_cells cells only the red children's residuals are evaluated (restrict_one<CW, 1>; option "restrict_red_cells")
// fold_first: the coarse level's first red half-sweep is stored by this kernel (restrict_one, cdinv); its down-stroke skips it
inline void plain_residual_restrict(vmg_s* h, int l, long long* count, bool after_black = false, bool fold_first = false)
{
    VmgLevel& L = h->lev[l];
    VmgLevel& C = h->lev[l + 1];
    C.cur = 0;
    C.first_red_done = fold_first;
    const double* cdinv = fold_first ? C.dinv : nullptr;
    dim3 grid, block;
    cell_launch_dims(C.G, grid, block);
    grid.z *= L.nprob;
    if (after_black && L.n >= h->restrict_red_cells) {
        launch_pdl(h, VMG_BY_WEIGHTS(L, residual_restrict_red_kernel), grid, block, 0, view(L), C.G, cur_phi(L), L.rhs, C.rhs, C.phi,
                   h->three_d ? 2 : 1, next_dir(h, L), cdinv);
    } else {
        launch_pdl(h, VMG_BY_WEIGHTS(L, residual_restrict_kernel), grid, block, 0, view(L), C.G, cur_phi(L), L.rhs, C.rhs, C.phi,
                   h->three_d ? 2 : 1, next_dir(h, L), cdinv);
    }
    ++*count;
}

inline ProlongBC prolong_bc(const vmg_s* h)
{
    ProlongBC bc;
    for (int f = 0; f < 6; ++f) bc.dirichlet[f] = h->bctype[f] == VMG_BC_DIRICHLET;
    return bc;
}

inline void plain_prolong_correct(vmg_s* h, int l, long long* count)
{
    VmgLevel& L = h->lev[l];
    if (h->prolong)
        launch_pdl(h, prolong_trilinear_kernel, grid_for(L.n), kThreads, 0, L.G, h->lev[l + 1].G, cur_phi(L), cur_phi(h->lev[l + 1]),
                   h->three_d ? 2 : 1, prolong_bc(h));
    else
        launch_pdl(h, prolong_correct_kernel, grid_for(L.n), kThreads, 0, L.G, h->lev[l + 1].G, cur_phi(L), cur_phi(h->lev[l + 1]),
                   h->three_d ? 2 : 1);
    ++*count;
}

// red_only: the level was last touched by a black half-sweep, after which the residual of every black cell is its own
// rounding error (rhs + s - fl(fl(dinv*(rhs + s))/dinv), ~2 ulp of D*phi, 1e-16 relative to ||btilde||): the norm is
// the maximum over the red cells, half the traffic (reading R12 in DESIGN.md).
inline void enqueue_residual_norm(vmg_s* h, unsigned long long* out, bool red_only = false, const unsigned long long* skip_if_zero = nullptr)
{
    VmgLevel& L = h->lev[0];
    dim3 grid, block;
    pair_launch_dims(L, grid, block);
    if (!red_only) grid.z *= 2;                               // one cell per thread: the planes once per colour
    const int zslots = (int)grid.z;
    if (skip_if_zero && L.nprob <= 1) grid.z = std::min(grid.z, 32u);   // vmg_solve's initial norm, which mostly skips itself
    ProfScope ps(h, VMG_PC_NORM, nullptr);
    if (L.cw == 0 && L.n >= h->phi_keep_cells)
        launch_pdl(h, residual_norm_kernel<0, 1>, grid, block, 0, view(L), cur_phi(L), L.rhs, out, next_dir(h, L), skip_if_zero, zslots);
    else
        launch_pdl(h, VMG_BY_WEIGHTS(L, residual_norm_kernel), grid, block, 0, view(L), cur_phi(L), L.rhs, out, next_dir(h, L), skip_if_zero, zslots);
}

// ------------------------------------------------------------------------------------------------
// S5: the coarse tail.  plan: the longest suffix of levels whose shared-memory blocks fit one CTA.
// ------------------------------------------------------------------------------------------------
constexpr size_t kTailSmemCap = 200 * 1024;

inline int tail_guard(const vmg_s* h, const VmgLevel& L) { return (h->three_d ? L.nx * L.ny : 0) + L.nx + 2; }

inline void plan_schedule(vmg_s* h)
{
    h->tail_level = -1;
    h->tail_smem = 0;
    if (!h->use_tail) return;
    size_t doubles = 0;
    int first = h->nlev;
    for (int l = h->nlev - 1; l >= 0 && h->nlev - l <= kTailMaxLevels; --l) {
        const VmgLevel& L = h->lev[l];
        if (L.n > 4096) break;
        size_t d = (size_t)tail_level_doubles((int)L.n, tail_guard(h, L));
        if ((doubles + d) * sizeof(double) > kTailSmemCap) break;
        doubles += d;
        first = l;
    }
    if (first == h->nlev) return;
    h->tail_level = first;
    h->tail_smem = doubles * sizeof(double);
    cudaFuncSetAttribute(coarse_tail_kernel<512>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kTailSmemCap);
    cudaFuncSetAttribute(coarse_tail_kernel<kTailThreads>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kTailSmemCap);
    // the level above the tail distributed over a thread-block cluster (vmg_cluster.cuh): z-slabs of P planes (P even), at
    // most 8 CTAs (the portable cluster size), one x-pair slot per thread, the slab's block beside the tail's in every CTA
    h->cl_nc = 0;
    const int d = first - 1;
    if (h->use_cluster && d >= 1 && h->three_d && !h->prolong) {
        const VmgLevel& D = h->lev[d];
        for (int nc = 8; nc >= 2; nc /= 2) {
            if (D.nz % (2 * nc)) continue;
            const int P = D.nz / nc;
            const long long nt = (long long)((D.nx + 1) / 2) * D.ny * P;
            const size_t bytes = (doubles + (size_t)tail_level_doubles(D.nx * D.ny * P, tail_guard(h, D))) * sizeof(double);
            if (nt > kTailThreads || bytes > kTailSmemCap) continue;
            h->cl_nc = nc; h->cl_P = P; h->cl_smem = bytes;
            h->tail_level = d;                       // the strokes hand levels >= d to enqueue_tail
            cudaFuncSetAttribute(coarse_cluster_kernel<512>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kTailSmemCap);
            cudaFuncSetAttribute(coarse_cluster_kernel<kTailThreads>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kTailSmemCap);
            break;
        }
    }
    (void)cudaGetLastError();
}

// launch with a thread-block cluster of nc CTAs (and programmatic stream serialisation like launch_pdl)
template <typename... KArgs, typename... Args>
inline void launch_cluster(vmg_s* h, void (*kernel)(KArgs...), unsigned grid, unsigned block, size_t smem, unsigned nc, Args... args)
{
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(block); cfg.dynamicSmemBytes = smem; cfg.stream = h->stream;
    cudaLaunchAttribute at[2];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = h->use_pdl ? 1 : 0;
    at[1].id = cudaLaunchAttributeClusterDimension;
    at[1].val.clusterDim.x = nc; at[1].val.clusterDim.y = 1; at[1].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 2;
    cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

inline void enqueue_tail(vmg_s* h, unsigned long long* norm_out, long long* count)
{
    TailArgs g;
    const bool clustered = h->cl_nc > 0;
    const int tail = h->tail_level + (clustered ? 1 : 0), first = tail;   // clustered: tail_level is the distributed level
    int off = 0;
    g.nl = h->nlev - first;
    for (int l = first; l < h->nlev; ++l) {
        VmgLevel& L = h->lev[l];
        TailLevel& T = g.lev[l - first];
        L.cur = 0;
        T.wx = L.wx; T.wy = L.wy; T.wz = L.wz; T.dinv = L.dinv; T.phi = L.phi; T.rhs = L.rhs;
        T.nx = L.nx; T.ny = L.ny; T.nz = L.nz; T.n = (int)L.n; T.nxy = L.nx * L.ny; T.G = L.G;
        T.zs = h->three_d ? T.nxy : 0;
        T.guard = tail_guard(h, L);
        T.off = off;
        if (l >= tail) off += tail_level_doubles(T.n, T.guard);
    }
    g.nu1 = h->nu1; g.nu2 = h->nu2; g.nbottom = h->nbottom; g.sz = h->three_d ? 2 : 1;
    g.prolong = h->prolong; g.bc = prolong_bc(h); g.sym = h->symmetric;
    g.whole = first == 0;
    g.norm_out = first == 0 ? norm_out : nullptr;
    g.pstride = h->lev[first].pstride;
    g.S = (h->use_bottom_matrix && h->lev[h->nlev - 1].n <= kBottomMatrixMax && h->nlev >= 2) ? h->bottom_S : nullptr;
    const int ncta = h->lev[first].nprob;
    ProfScope ps(h, VMG_PC_COARSE, count);
    if (clustered) {
        ClusterArgs c;
        c.tail = g;
        VmgLevel& L = h->lev[first - 1];
        TailLevel& T = c.D;
        L.cur = 0;
        T.wx = L.wx; T.wy = L.wy; T.wz = L.wz; T.dinv = L.dinv; T.phi = L.phi; T.rhs = L.rhs;
        T.nx = L.nx; T.ny = L.ny; T.nz = L.nz; T.n = (int)L.n; T.nxy = L.nx * L.ny; T.G = L.G;
        T.zs = T.nxy;
        T.guard = tail_guard(h, L);
        T.off = off;                                  // behind the tail's levels
        c.P = h->cl_P;
        const long long nt = (long long)((L.nx + 1) / 2) * L.ny * h->cl_P;
        int threads = (int)std::max<long long>((nt + 31) / 32 * 32, std::min<long long>(kTailThreads, std::max<long long>(64, (h->lev[first].n / 2 + 31) / 32 * 32)));
        if (threads <= 512) launch_cluster(h, coarse_cluster_kernel<512>, (unsigned)(ncta * h->cl_nc), (unsigned)threads, h->cl_smem, (unsigned)h->cl_nc, c);
        else launch_cluster(h, coarse_cluster_kernel<kTailThreads>, (unsigned)(ncta * h->cl_nc), (unsigned)threads, h->cl_smem, (unsigned)h->cl_nc, c);
    } else
    {
        int threads = (int)std::min<long long>(kTailThreads, std::max<long long>(64, (h->lev[first].n / 2 + 31) / 32 * 32));
        if (threads <= 512) launch_pdl(h, coarse_tail_kernel<512>, ncta, threads, h->tail_smem, g);
        else launch_pdl(h, coarse_tail_kernel<kTailThreads>, ncta, threads, h->tail_smem, g);
    }
    ++*count;
}

// ------------------------------------------------------------------------------------------------
// S2-S4, S6: blocked passes.  Tile width 40 (32 interior + 2 x 4 halo); one thread per 2 x 2 patch, at most 384
// threads (168 registers each), the tile height is the largest even number of rows that fits threads and shared memory.
// ------------------------------------------------------------------------------------------------
constexpr int kBlkNXT = 40;
constexpr int kBlkMaxSmem = 232448 - 1024;
constexpr int kBlkMaxThreads = 384;

constexpr int blk_pick_nyt(int S, int TAIL)
{
    int best = 0;
    for (int nyt = 2 * (S + 2) + 2; nyt <= 64; nyt += 2) {
        long long nph = (long long)(kBlkNXT / 2) * (nyt / 2);
        int rs = S + (TAIL ? 1 : 0);
        long long smem = (long long)rs * 20 * nph * 8;
        if (nph <= kBlkMaxThreads && smem <= kBlkMaxSmem) best = nyt;
    }
    return best;
}

template <int S, int TAIL, bool PROLONG, int C0>
struct BlkKernel {
    static constexpr int NYT = blk_pick_nyt(S, TAIL);
    using C = BlockCfg<S, TAIL, kBlkNXT, NYT>;
    static void prepare()
    {
        cudaFuncSetAttribute(smooth_block_kernel<S, TAIL, PROLONG, C0, kBlkNXT, NYT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)C::SMEM);
    }
    static void launch(vmg_s* h, BlockArgs g)
    {
        g.ntx = (int)cdiv(g.G.nx, C::TX); g.nty = (int)cdiv(g.G.ny, C::TY);
        // z-segments per tile: minimise waves x (planes per CTA incl. the 2H halo planes each segment pays)
        const long long ntiles = (long long)g.ntx * g.nty;
        int best = 1;
        double best_cost = 1e300;
        for (int ns = 1; ns <= std::max(1, g.G.nz / 4); ++ns) {
            double waves = (double)cdiv(ntiles * ns, h->num_sms);
            double cost = waves * ((double)cdiv(g.G.nz / 2, ns) * 2 + 2 * C::H + 2);
            if (cost < best_cost) { best_cost = cost; best = ns; }
        }
        g.nzseg = best;
        unsigned grid = (unsigned)(ntiles * g.nzseg);
        smooth_block_kernel<S, TAIL, PROLONG, C0, kBlkNXT, NYT><<<grid, C::NT, C::SMEM, h->stream>>>(g);
    }
};

#define VMG_BLK_CASE(S_, T_, P_)                                                             \
    if (prepare_all) { BlkKernel<S_, T_, P_, 0>::prepare(); BlkKernel<S_, T_, P_, 1>::prepare(); } \
    else if (S == S_ && tail == T_ && prolong == P_) {                                       \
        if (g.colour0 & 1) BlkKernel<S_, T_, P_, 1>::launch(h, g); else BlkKernel<S_, T_, P_, 0>::launch(h, g); \
        return;                                                                              \
    }

inline void blk_run(vmg_s* h, const BlockArgs& g, int S, int tail, bool prolong, bool prepare_all = false)
{
    VMG_BLK_CASE(1, 0, false) VMG_BLK_CASE(1, 0, true) VMG_BLK_CASE(1, 1, false) VMG_BLK_CASE(1, 1, true)
    VMG_BLK_CASE(1, 2, false) VMG_BLK_CASE(1, 2, true)
    VMG_BLK_CASE(2, 0, false) VMG_BLK_CASE(2, 0, true) VMG_BLK_CASE(2, 1, false) VMG_BLK_CASE(2, 1, true)
    VMG_BLK_CASE(2, 2, false) VMG_BLK_CASE(2, 2, true)
    VMG_BLK_CASE(3, 0, false) VMG_BLK_CASE(3, 0, true) VMG_BLK_CASE(3, 1, false) VMG_BLK_CASE(3, 1, true)
    VMG_BLK_CASE(3, 2, false) VMG_BLK_CASE(3, 2, true)
}
#undef VMG_BLK_CASE

// ------------------------------------------------------------------------------------------------
// S2-S4, S6: blocked passes, third design (vmg_block3.cuh; option blocked = 2): TMA-fed ring, one split barrier per plane.
// ------------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// cuTensorMapEncodeTiled through the runtime's driver entry point: the library does not link libcuda
inline EncodeTiledFn tensor_map_encoder()
{
    static EncodeTiledFn fn = nullptr;
    static std::once_flag once;
    std::call_once(once, [] {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
        (void)cudaGetLastError();
    });
    return fn;
}

// A level array (x-parity split rows, Geom) as the 5-D fp64 tensor (m, row pair, row parity, x-parity, plane); a box
// {nxp, nyt/2, 2, 2, 1} lands in shared memory as [x-parity][row parity][row pair][m].  ny must be even.
inline bool make_level_tensor_map(CUtensorMap* map, const Geom& G, const double* base, int nxp, int nyt)
{
    EncodeTiledFn enc = tensor_map_encoder();
    if (!enc) return false;
    const cuuint64_t dims[5] = {(cuuint64_t)G.hp, (cuuint64_t)(G.ny / 2), 2, 2, (cuuint64_t)G.nz};
    const cuuint64_t strides[4] = {(cuuint64_t)2 * G.pitch * 8, (cuuint64_t)G.pitch * 8, (cuuint64_t)G.hp * 8, (cuuint64_t)G.plane * 8};
    const cuuint32_t box[5] = {(cuuint32_t)nxp, (cuuint32_t)(nyt / 2), 2, 2, 1};
    const cuuint32_t es[5] = {1, 1, 1, 1, 1};
    return enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 5, (void*)base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// the same array as the 4-D tensor (m, row, x-parity, plane): a box {nxp, nyt, 2, 1} lands as [x-parity][row][m] (row variant)
inline bool make_level_tensor_map4(CUtensorMap* map, const Geom& G, const double* base, int nxp, int nyt)
{
    EncodeTiledFn enc = tensor_map_encoder();
    if (!enc) return false;
    const cuuint64_t dims[4] = {(cuuint64_t)G.hp, (cuuint64_t)G.ny, 2, (cuuint64_t)G.nz};
    const cuuint64_t strides[3] = {(cuuint64_t)G.pitch * 8, (cuuint64_t)G.hp * 8, (cuuint64_t)G.plane * 8};
    const cuuint32_t box[4] = {(cuuint32_t)nxp, (cuuint32_t)nyt, 2, 1};
    const cuuint32_t es[4] = {1, 1, 1, 1};
    return enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, (void*)base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// the level's tensor maps are encoded once per (array, box) and kept with the level
inline bool level_map(VmgLevel& L, const double* base, int nxp, int nyt, CUtensorMap* out, int rank = 5)
{
    for (auto& m : L.tmaps)
        if (m.base == base && m.nxp == nxp && m.nyt == nyt && m.rank == rank) { *out = m.map; return true; }
    VmgTensorMap m;
    m.base = base; m.nxp = nxp; m.nyt = nyt; m.rank = rank;
    if (!(rank == 5 ? make_level_tensor_map(&m.map, L.G, base, nxp, nyt) : make_level_tensor_map4(&m.map, L.G, base, nxp, nyt))) return false;
    L.tmaps.push_back(m);
    *out = m.map;
    return true;
}

constexpr int kB3NXT = 40;
constexpr int kB3PF = 1;
constexpr int kB3MaxSmem = 232448;
constexpr int kB3MaxThreads = 384;

constexpr int b3_pick_nyt(int S, int T)
{
    int best = 0;
    for (int nyt = 10; nyt <= 64; nyt += 2) {
        const long long nph = (long long)(kB3NXT / 2) * (nyt / 2);
        const int ns = S + T + 1 + kB3PF, np = S + T;
        const long long smem = (long long)(3 * ns + 2 * np) * 4 * nph * 8 + (ns + 1) * 8 + 128;
        if (nph <= kB3MaxThreads && smem <= kB3MaxSmem) best = nyt;
    }
    return best;
}

template <int S, int TAIL, bool PROLONG, int C0>
struct B3Kernel {
    static constexpr int NYT = b3_pick_nyt(S, TAIL ? 1 : 0);
    using C = B3Cfg<S, TAIL, kB3NXT, NYT, kB3PF>;
    static void prepare()
    {
        cudaFuncSetAttribute(smooth_block3_kernel<S, TAIL, PROLONG, C0, kB3NXT, NYT, kB3PF>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)C::SMEM);
    }
    static bool launch(vmg_s* h, VmgLevel& L, Block3Args& g, const double* phi_in)
    {
        if (!level_map(L, phi_in, C::NXP, NYT, &g.tm_phi) || !level_map(L, L.wx, C::NXP, NYT, &g.tm_wx) ||
            !level_map(L, L.wy, C::NXP, NYT, &g.tm_wy))
            return false;
        g.ntx = (int)cdiv(g.G.nx, C::TX); g.nty = (int)cdiv(g.G.ny, C::TY);
        // z-segments per tile: minimise waves x (planes per CTA incl. the 2 ZH halo planes each segment pays)
        const long long ntiles = (long long)g.ntx * g.nty;
        int best = 1;
        double best_cost = 1e300;
        for (int ns = 1; ns <= std::max(1, g.G.nz / 4); ++ns) {
            double waves = (double)cdiv(ntiles * ns, h->num_sms);
            double cost = waves * ((double)cdiv(g.G.nz / 2, ns) * 2 + 2 * C::ZH + 2);
            if (cost < best_cost) { best_cost = cost; best = ns; }
        }
        g.nzseg = best;
        unsigned grid = (unsigned)(ntiles * g.nzseg);
        smooth_block3_kernel<S, TAIL, PROLONG, C0, kB3NXT, NYT, kB3PF><<<grid, C::NT, C::SMEM, h->stream>>>(g);
        return true;
    }
};

#define VMG_B3_CASE(S_, T_, P_)                                                              \
    if (prepare_all) { B3Kernel<S_, T_, P_, 0>::prepare(); B3Kernel<S_, T_, P_, 1>::prepare(); } \
    else if (S == S_ && tail == T_ && prolong == P_)                                         \
        return (g.colour0 & 1) ? B3Kernel<S_, T_, P_, 1>::launch(h, *L, g, phi_in) : B3Kernel<S_, T_, P_, 0>::launch(h, *L, g, phi_in);

inline bool b3_run(vmg_s* h, VmgLevel* L, Block3Args& g, const double* phi_in, int S, int tail, bool prolong, bool prepare_all = false)
{
    VMG_B3_CASE(1, 0, false) VMG_B3_CASE(1, 0, true) VMG_B3_CASE(1, 1, false) VMG_B3_CASE(1, 1, true)
    VMG_B3_CASE(1, 2, false) VMG_B3_CASE(1, 2, true)
    VMG_B3_CASE(2, 0, false) VMG_B3_CASE(2, 0, true) VMG_B3_CASE(2, 1, false) VMG_B3_CASE(2, 1, true)
    VMG_B3_CASE(2, 2, false) VMG_B3_CASE(2, 2, true)
    VMG_B3_CASE(3, 0, false) VMG_B3_CASE(3, 0, true) VMG_B3_CASE(3, 1, false) VMG_B3_CASE(3, 1, true)
    VMG_B3_CASE(3, 2, false) VMG_B3_CASE(3, 2, true)
    return prepare_all;
}
#undef VMG_B3_CASE

// row variant (option blocked = 3): one thread per x-pair of one row, up to 704 threads
constexpr int kB3rMaxThreads = 704;
constexpr int b3r_pick_nyt(int S, int TAIL)
{
    const int T = TAIL ? 1 : 0;
    int best = 0;
    for (int nyt = 2 * (S + T) + 2; nyt <= 64; nyt += 2) {
        const long long nph = (long long)(kB3NXT / 2) * nyt;
        const int ns = S + T + 1 + kB3PF, np = S + T;
        const long long smem = ((long long)(3 * ns + 2 * np) * 2 * nph + (TAIL == BT_RESTRICT ? 2 * nph : 0)) * 8 + 256;
        if (nph <= kB3rMaxThreads && smem <= kB3MaxSmem) best = nyt;
    }
    return best;
}

template <int S, int TAIL, bool PROLONG, int C0>
struct B3rKernel {
    static constexpr int NYT = b3r_pick_nyt(S, TAIL);
    using C = B3rCfg<S, TAIL, kB3NXT, NYT, kB3PF>;
    static void prepare()
    {
        cudaFuncSetAttribute(smooth_block3r_kernel<S, TAIL, PROLONG, C0, kB3NXT, NYT, kB3PF>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)C::SMEM);
    }
    static bool launch(vmg_s* h, VmgLevel& L, Block3Args& g, const double* phi_in)
    {
        if (!level_map(L, phi_in, C::NXP, NYT, &g.tm_phi, 4) || !level_map(L, L.wx, C::NXP, NYT, &g.tm_wx, 4) ||
            !level_map(L, L.wy, C::NXP, NYT, &g.tm_wy, 4))
            return false;
        g.ntx = (int)cdiv(g.G.nx, C::TX); g.nty = (int)cdiv(g.G.ny, C::TY);
        const long long ntiles = (long long)g.ntx * g.nty;
        int best = 1;
        double best_cost = 1e300;
        for (int ns = 1; ns <= std::max(1, g.G.nz / 4); ++ns) {
            double waves = (double)cdiv(ntiles * ns, h->num_sms);
            double cost = waves * ((double)cdiv(g.G.nz / 2, ns) * 2 + 2 * C::ZH + 2);
            if (cost < best_cost) { best_cost = cost; best = ns; }
        }
        g.nzseg = best;
        unsigned grid = (unsigned)(ntiles * g.nzseg);
        smooth_block3r_kernel<S, TAIL, PROLONG, C0, kB3NXT, NYT, kB3PF><<<grid, C::NT, C::SMEM, h->stream>>>(g);
        return true;
    }
};

#define VMG_B3R_CASE(S_, T_, P_)                                                             \
    if (prepare_all) { B3rKernel<S_, T_, P_, 0>::prepare(); B3rKernel<S_, T_, P_, 1>::prepare(); } \
    else if (S == S_ && tail == T_ && prolong == P_)                                         \
        return (g.colour0 & 1) ? B3rKernel<S_, T_, P_, 1>::launch(h, *L, g, phi_in) : B3rKernel<S_, T_, P_, 0>::launch(h, *L, g, phi_in);

inline bool b3r_run(vmg_s* h, VmgLevel* L, Block3Args& g, const double* phi_in, int S, int tail, bool prolong, bool prepare_all = false)
{
    VMG_B3R_CASE(1, 0, false) VMG_B3R_CASE(1, 0, true) VMG_B3R_CASE(1, 1, false) VMG_B3R_CASE(1, 1, true)
    VMG_B3R_CASE(1, 2, false) VMG_B3R_CASE(1, 2, true)
    VMG_B3R_CASE(2, 0, false) VMG_B3R_CASE(2, 0, true) VMG_B3R_CASE(2, 1, false) VMG_B3R_CASE(2, 1, true)
    VMG_B3R_CASE(2, 2, false) VMG_B3R_CASE(2, 2, true)
    VMG_B3R_CASE(3, 0, false) VMG_B3R_CASE(3, 0, true) VMG_B3R_CASE(3, 1, false) VMG_B3R_CASE(3, 1, true)
    VMG_B3R_CASE(3, 2, false) VMG_B3R_CASE(3, 2, true)
    return prepare_all;
}
#undef VMG_B3R_CASE

// once per process, outside any stream capture
inline void prepare_blocked(vmg_s* h)
{
    static std::once_flag once[64];   // per device: the attributes belong to the device's copy of the kernels
    std::call_once(once[h->device & 63], [&] {
        BlockArgs g{};
        blk_run(h, g, 0, 0, false, true);
        Block3Args g3{};
        b3_run(h, nullptr, g3, nullptr, 0, 0, false, true);
        b3r_run(h, nullptr, g3, nullptr, 0, 0, false, true);
        (void)cudaGetLastError();
    });
}

inline bool blocked_ok(const vmg_s* h, int l)
{
    const VmgLevel& L = h->lev[l];
    return h->use_blocked && h->three_d && L.nx % 2 == 0 && L.ny % 2 == 0 && L.nz % 2 == 0 && L.n >= h->block_min_cells;
}

// nhalf colour half-sweeps starting with colour `colour0` on level l, as ceil(nhalf/3) blocked passes; the first
// pass may add the coarse correction while loading (prolong), the last may end with a residual stage (tail).
inline void blocked_sweeps(vmg_s* h, int l, int nhalf, int colour0, bool prolong, int tail, unsigned long long* norm_out,
                           long long* count)
{
    VmgLevel& L = h->lev[l];
    int passes = (nhalf + 2) / 3, base = nhalf / passes, rem = nhalf % passes, done = 0;
    for (int p = 0; p < passes; ++p) {
        int S = base + (p < rem ? 1 : 0);
        BlockArgs g{};
        g.wx = L.wx; g.wy = L.wy; g.wz = L.wz; g.dinv = L.dinv; g.rhs = L.rhs;
        g.phi_in = cur_phi(L); g.phi_out = other_phi(L);
        g.G = L.G;
        g.colour0 = (colour0 + done) & 1;
        bool first = p == 0, last = p == passes - 1;
        int T = last ? tail : BT_NONE;
        if ((first && prolong) || T == BT_RESTRICT) {
            VmgLevel& C = h->lev[l + 1];
            g.CG = C.G;
            if (first && prolong) g.e = cur_phi(C);
            if (T == BT_RESTRICT) { C.cur = 0; g.crhs = C.rhs; g.cphi = C.phi; }
        }
        g.norm_out = norm_out;
        if (h->use_blocked >= 2) {
            Block3Args g3{};
            g3.wz = L.wz; g3.dinv = L.dinv; g3.rhs = L.rhs; g3.phi_out = g.phi_out;
            g3.G = g.G; g3.CG = g.CG; g3.colour0 = g.colour0; g3.e = g.e; g3.crhs = g.crhs; g3.cphi = g.cphi; g3.norm_out = norm_out;
            const bool okl = h->use_blocked == 3 ? b3r_run(h, &L, g3, g.phi_in, S, T, first && prolong)
                                                 : b3_run(h, &L, g3, g.phi_in, S, T, first && prolong);
            if (!okl) h->last_cuda_error = (int)cudaErrorNotSupported;
        } else
        blk_run(h, g, S, T, first && prolong);
        L.cur ^= 1;
        done += S;
        ++*count;
    }
}

// leaves phi of level l in its primary buffer
inline void settle_phi(vmg_s* h, int l)
{
    VmgLevel& L = h->lev[l];
    if (L.cur == 0) return;
    cudaMemcpyAsync(L.phi, L.phi2, L.nalloc * sizeof(double), cudaMemcpyDeviceToDevice, h->stream);
    L.cur = 0;
}

// nsweeps red-black sweeps on the level's phi (primary buffer in, primary buffer out)
inline void enqueue_smooth(vmg_s* h, int l, int nsweeps, long long* count)
{
    ProfScope ps(h, l == 0 ? VMG_PC_SMOOTH0 : VMG_PC_COARSE, count);
    h->lev[l].cur = 0;
    if (nsweeps > 0 && blocked_ok(h, l)) {
        blocked_sweeps(h, l, 2 * nsweeps, 0, false, BT_NONE, nullptr, count);
        settle_phi(h, l);
    } else {
        plain_smooth(h, l, nsweeps, count);
    }
}

// Can the restriction INTO level c store that level's first red half-sweep (plain_residual_restrict fold_first)?  Only when
// level c runs an ordinary down-stroke of per-colour launches afterwards: not the tail / bottom level, not a blocked level.
inline bool can_fold_first(const vmg_s* h, int c)
{
    const int last = h->nlev - 1;
    const int tail = h->tail_level < 0 ? last : h->tail_level;
    return h->nu1 >= 1 && c < tail && !blocked_ok(h, c);
}

// down-stroke of level l: nu1 sweeps then residual+restriction into level l+1 (which also zeroes its phi)
// chain: part of a whole V-cycle (the next level's down-stroke follows): the restriction may store the next level's first
// red half-sweep; a single stroke (vmg_step_down) never does
inline void enqueue_down(vmg_s* h, int l, long long* count, bool chain = false)
{
    VmgLevel& L = h->lev[l];
    const int skip = L.first_red_done ? 1 : 0;
    L.first_red_done = false;
    if (h->nu1 > 0 && blocked_ok(h, l)) {
        ProfScope ps(h, l == 0 ? VMG_PC_SMOOTH0 : VMG_PC_COARSE, count);
        blocked_sweeps(h, l, 2 * h->nu1, 0, false, BT_RESTRICT, nullptr, count);
        return;
    }
    {
        ProfScope ps(h, l == 0 ? VMG_PC_SMOOTH0 : VMG_PC_COARSE, count);
        plain_smooth(h, l, h->nu1, count, skip);
    }
    ProfScope ps(h, l == 0 ? VMG_PC_RESREST0 : VMG_PC_COARSE, count);
    plain_residual_restrict(h, l, count, h->nu1 >= 1, chain && can_fold_first(h, l + 1));
}

// up-stroke of level l: prolongation+correction from level l+1 then nu2 sweeps [then the residual norm (level 0)].
// Returns true if the residual norm was fused into the stroke.
inline bool enqueue_up(vmg_s* h, int l, unsigned long long* norm_out, long long* count)
{
    if (h->nu2 > 0 && blocked_ok(h, l)) {
        if (h->prolong) {   // the blocked passes can only add a piecewise-constant correction while loading
            ProfScope ps(h, l == 0 ? VMG_PC_PROLONG0 : VMG_PC_COARSE, count);
            plain_prolong_correct(h, l, count);
        }
        ProfScope ps(h, l == 0 ? VMG_PC_SMOOTH0 : VMG_PC_COARSE, count);
        bool fuse = l == 0 && norm_out != nullptr;
        blocked_sweeps(h, l, 2 * h->nu2, h->symmetric, !h->prolong, fuse ? BT_NORM : BT_NONE, norm_out, count);
        return fuse;
    }
    if (h->nu2 >= 1 && !h->prolong) {   // the correction rides on the first half-sweep (smooth_colour_prolong_kernel)
        ProfScope ps(h, l == 0 ? VMG_PC_SMOOTH0 : VMG_PC_COARSE, count);
        VmgLevel& L = h->lev[l];
        dim3 grid, block;
        pair_launch_dims(L, grid, block);
        if (L.cw == 0 && L.n >= h->phi_keep_cells)
            launch_pdl(h, smooth_colour_prolong_kernel<0, 1>, grid, block, 0, view(L), h->lev[l + 1].G, cur_phi(L), L.rhs,
                       cur_phi(h->lev[l + 1]), h->symmetric, h->three_d ? 2 : 1, next_dir(h, L));
        else
            launch_pdl(h, VMG_BY_WEIGHTS(L, smooth_colour_prolong_kernel), grid, block, 0, view(L), h->lev[l + 1].G, cur_phi(L), L.rhs,
                       cur_phi(h->lev[l + 1]), h->symmetric, h->three_d ? 2 : 1, next_dir(h, L));
        ++*count;
        plain_smooth(h, l, h->nu2, count, 1, h->symmetric);
        return false;
    }
    {
        ProfScope ps(h, l == 0 ? VMG_PC_PROLONG0 : VMG_PC_COARSE, count);
        plain_prolong_correct(h, l, count);
    }
    ProfScope ps(h, l == 0 ? VMG_PC_SMOOTH0 : VMG_PC_COARSE, count);
    plain_smooth(h, l, h->nu2, count, 0, h->symmetric);
    return false;
}

// C4: one V-cycle on the handle's own level arrays (level-0 phi / rhs = btilde already in place, primary buffer).
// If norm_out is given, *norm_out (zeroed here) receives the bit pattern of ||rhs - A phi||_inf on level 0.
inline void enqueue_vcycle(vmg_s* h, unsigned long long* norm_out, long long* count)
{
    const int last = h->nlev - 1;
    // first level not handled stroke by stroke
    const int tail = h->tail_level < 0 ? last : h->tail_level;
    if (norm_out) cudaMemsetAsync(norm_out, 0, sizeof(unsigned long long), h->stream);
    for (int l = 0; l <= last; ++l) { h->lev[l].cur = 0; h->lev[l].dir = 0; h->lev[l].first_red_done = false; }
    for (int l = 0; l < tail; ++l) enqueue_down(h, l, count, true);
    bool norm_done = false;
    if (h->tail_level >= 0) {
        enqueue_tail(h, norm_out, count);
        norm_done = h->tail_level == 0 && norm_out;
    } else {
        VmgLevel& B = h->lev[last];
        if (last == 0) cudaMemsetAsync(B.phi, 0, B.nalloc * sizeof(double), h->stream);   // single level: bottom from zero
        ProfScope ps(h, VMG_PC_COARSE, count);
        if (!h->symmetric) plain_smooth(h, last, h->nbottom, count);
        else { plain_smooth(h, last, h->nbottom / 2, count, 0, 0); plain_smooth(h, last, h->nbottom - h->nbottom / 2, count, 0, 1); }
    }
    for (int l = tail - 1; l >= 0; --l) norm_done = enqueue_up(h, l, l == 0 ? norm_out : nullptr, count);
    if (norm_out && !norm_done) { enqueue_residual_norm(h, norm_out, h->nu2 >= 1 && tail > 0 && !h->symmetric); ++*count; }
    settle_phi(h, 0);
}

// The same cycle in three pieces (staggered batch schedule of vmg_solve_batch): 0 = level-0 down-stroke, 1 = all coarser
// levels (strokes of levels 1.., tail or bottom solve), 2 = level-0 up-stroke + residual norm.  Enqueued in this order they
// are enqueue_vcycle, launch for launch.
inline bool vcycle_segmentable(const vmg_s* h)
{
    const int last = h->nlev - 1;
    const int tail = h->tail_level < 0 ? last : h->tail_level;
    return tail >= 1 && h->use_graph && !h->profile;
}

inline void enqueue_vcycle_segment(vmg_s* h, int seg, unsigned long long* norm_out, long long* count)
{
    const int last = h->nlev - 1;
    const int tail = h->tail_level < 0 ? last : h->tail_level;
    if (seg == 0) {
        cudaMemsetAsync(norm_out, 0, sizeof(unsigned long long), h->stream);
        for (int l = 0; l <= last; ++l) { h->lev[l].cur = 0; h->lev[l].dir = 0; h->lev[l].first_red_done = false; }
        enqueue_down(h, 0, count, true);
    } else if (seg == 1) {
        for (int l = 1; l < tail; ++l) enqueue_down(h, l, count, true);
        if (h->tail_level >= 0) enqueue_tail(h, nullptr, count);
        else {
            ProfScope ps(h, VMG_PC_COARSE, count);
            if (!h->symmetric) plain_smooth(h, last, h->nbottom, count);
            else { plain_smooth(h, last, h->nbottom / 2, count, 0, 0); plain_smooth(h, last, h->nbottom - h->nbottom / 2, count, 0, 1); }
        }
        for (int l = tail - 1; l >= 1; --l) enqueue_up(h, l, nullptr, count);
    } else {
        const bool norm_done = enqueue_up(h, 0, norm_out, count);
        if (!norm_done) { enqueue_residual_norm(h, norm_out, h->nu2 >= 1 && !h->symmetric); ++*count; }
        settle_phi(h, 0);
    }
}

// Members of a vmg_create_batch group share one stream, and the access-policy window that keeps a handle's level-0 face
// weights in L2 is a stream attribute which captured kernel nodes inherit: before a member captures, it puts ITS window
// back on the stream (otherwise every member's graph would carry the window of whichever member was prepared last).
inline void own_l2_window(vmg_s* h)
{
    if (h->group && h->l2_window_set) {
        cudaStreamSetAttribute(h->stream, cudaStreamAttributeAccessPolicyWindow, &h->l2_attr);
        (void)cudaGetLastError();
    }
}

// captures the three segments (once per epoch and kind of weights), then launches segment `seg` into `into`
// (the handle's stream, or its high-priority stream for segment 1: a graph runs at the priority of the stream it is
// launched into)
inline int run_vcycle_segment(vmg_s* h, int seg, unsigned long long* out, cudaStream_t into = nullptr)
{
    const int gi = h->lev[0].cw;
    if (h->seg_epoch[gi] != h->graph_epoch) {
        prepare_blocked(h);
        own_l2_window(h);
        for (int sg = 0; sg < 3; ++sg) {
            if (h->seg_exec[gi][sg]) { cudaGraphExecDestroy(h->seg_exec[gi][sg]); h->seg_exec[gi][sg] = nullptr; }
            if (h->seg_graph[gi][sg]) { cudaGraphDestroy(h->seg_graph[gi][sg]); h->seg_graph[gi][sg] = nullptr; }
            long long count = 0;
            if (cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeRelaxed) != cudaSuccess) {
                h->last_cuda_error = (int)cudaGetLastError();
                return VMG_ERR_CUDA;
            }
            enqueue_vcycle_segment(h, sg, out, &count);
            cudaError_t e = cudaStreamEndCapture(h->stream, &h->seg_graph[gi][sg]);
            if (e == cudaSuccess) e = cudaGraphInstantiate(&h->seg_exec[gi][sg], h->seg_graph[gi][sg], 0);
            if (e != cudaSuccess) { h->last_cuda_error = (int)e; (void)cudaGetLastError(); return VMG_ERR_CUDA; }
            h->seg_launches[gi][sg] = count;
        }
        h->seg_epoch[gi] = h->graph_epoch;
    }
    cudaError_t e = cudaGraphLaunch(h->seg_exec[gi][seg], into ? into : h->stream);
    if (e != cudaSuccess) { h->last_cuda_error = (int)e; (void)cudaGetLastError(); return VMG_ERR_CUDA; }
    h->launches += h->seg_launches[gi][seg];
    if (seg == 2) h->launches_per_cycle = h->seg_launches[gi][0] + h->seg_launches[gi][1] + h->seg_launches[gi][2];
    return VMG_OK;
}

// ------------------------------------------------------------------------------------------------
// S7 with the convergence test on the device ("device-side WHILE conditional node") and the
// residual norm fused into the next cycle (S6 "0 (fused)").  One graph per solve:
//     head:   norm accumulator = 0;  H1 = red half-sweep of cycle 1: neighbours from phi, red cells -> phi2
//     WHILE (continue) {
//         black half-sweep: (red) neighbours from phi2, black cells -> phi;   rest of the cycle in place on phi
//         H1 of the NEXT cycle, which also takes the red-cell residual norm of the iterate just completed (reading R12)
//         solve_decide_kernel: history, exit rules C5, sets `continue`
//     }
// phi itself holds the completed iterate until the device has decided to go on, so a converged solve returns exactly
// the iterate the host-driven loop returns (bitwise: same kernels' arithmetic, same norms); what it costs is one red
// half-sweep after the last cycle (21 us on config 3) in place of a residual-norm kernel per cycle (30 us) and of the
// host round trip between cycles.
// ------------------------------------------------------------------------------------------------
inline bool solve_loop_ok(vmg_s* h, int max_vcycles)
{
    const int last = h->nlev - 1;
    const int tail = h->tail_level < 0 ? last : h->tail_level;
    // nu1 >= 2: the red cells relaxed by H1 live in phi2 until the second red half-sweep of the down-stroke rewrites them in phi
    return h->use_loop && h->use_graph && !h->profile && h->nu1 >= 2 && h->nu2 >= 1 && !h->symmetric && tail >= 1 &&
           !blocked_ok(h, 0) && max_vcycles >= 1 && max_vcycles <= kLoopMaxCycles;
}

// a colour half-sweep of level 0 with separate input / output arrays, optionally with the norm of the cells it relaxes
inline void loop_halfsweep_io(vmg_s* h, const double* in, double* out, int colour, bool norm, unsigned long long* norm_out, long long* count)
{
    VmgLevel& L = h->lev[0];
    LevelView v = view(L);
    dim3 grid, block;
    pair_launch_dims(L, grid, block);
    const int dir = next_dir(h, L);
    const bool keep = L.cw == 0 && L.n >= h->phi_keep_cells;
#define VMG_IO(CW_, KEEP_) (norm ? smooth_colour_io_kernel<CW_, KEEP_, 1> : smooth_colour_io_kernel<CW_, KEEP_, 0>)
    auto kernel = L.cw == 2 ? VMG_IO(2, 0) : L.cw == 1 ? VMG_IO(1, 0) : keep ? VMG_IO(0, 1) : VMG_IO(0, 0);
#undef VMG_IO
    launch_pdl(h, kernel, grid, block, 0, v, in, out, L.rhs, colour, dir, norm_out);
    ++*count;
}

// one WHILE iteration (see above); the levels' phi in their primary buffers
inline void enqueue_loop_body(vmg_s* h, cudaGraphConditionalHandle handle, unsigned long long* norm_out, long long* count)
{
    const int last = h->nlev - 1;
    const int tail = h->tail_level < 0 ? last : h->tail_level;
    for (int l = 0; l <= last; ++l) { h->lev[l].cur = 0; h->lev[l].dir = 0; h->lev[l].first_red_done = false; }
    VmgLevel& L0 = h->lev[0];
    L0.dir = 1;                                                   // the half-sweep before this one walked forward
    loop_halfsweep_io(h, L0.phi2, L0.phi, 1, false, nullptr, count);
    plain_smooth(h, 0, h->nu1, count, 2);
    plain_residual_restrict(h, 0, count, true, can_fold_first(h, 1));
    for (int l = 1; l < tail; ++l) enqueue_down(h, l, count, true);
    if (h->tail_level >= 0) enqueue_tail(h, nullptr, count);
    else {
        if (!h->symmetric) plain_smooth(h, last, h->nbottom, count);
        else { plain_smooth(h, last, h->nbottom / 2, count, 0, 0); plain_smooth(h, last, h->nbottom - h->nbottom / 2, count, 0, 1); }
    }
    for (int l = tail - 1; l >= 0; --l) enqueue_up(h, l, nullptr, count);
    loop_halfsweep_io(h, L0.phi, L0.phi2, 0, true, norm_out, count);
    solve_decide_kernel<<<1, 32, 0, h->stream>>>(handle, h->d_loop, norm_out);
    ++*count;
}

// builds (once per epoch and kind of weights) and launches the solve graph; the caller has filled h->h_loop[0..8]
inline int run_solve_loop(vmg_s* h, unsigned long long* norm_out)
{
    const int gi = h->lev[0].cw;
    auto fail = [&](cudaError_t e) { h->last_cuda_error = (int)e; (void)cudaGetLastError(); return VMG_ERR_CUDA; };
    if (h->loop_epoch[gi] != h->graph_epoch) {
        own_l2_window(h);
        if (h->loop_exec[gi]) { cudaGraphExecDestroy(h->loop_exec[gi]); h->loop_exec[gi] = nullptr; }
        if (h->loop_graph[gi]) { cudaGraphDestroy(h->loop_graph[gi]); h->loop_graph[gi] = nullptr; }
        cudaGraph_t g = nullptr, dummy = nullptr;
        cudaError_t e = cudaGraphCreate(&g, 0);
        if (e != cudaSuccess) return fail(e);
        h->loop_graph[gi] = g;
        cudaGraphConditionalHandle handle;
        if ((e = cudaGraphConditionalHandleCreate(&handle, g, 1, cudaGraphCondAssignDefault)) != cudaSuccess) return fail(e);
        // head
        long long count = 0;
        if ((e = cudaStreamBeginCaptureToGraph(h->stream, g, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed)) != cudaSuccess) return fail(e);
        cudaMemsetAsync(norm_out, 0, sizeof(unsigned long long), h->stream);
        for (int l = 0; l < h->nlev; ++l) { h->lev[l].cur = 0; h->lev[l].dir = 0; }
        loop_halfsweep_io(h, h->lev[0].phi, h->lev[0].phi2, 0, false, nullptr, &count);
        cudaStreamCaptureStatus st;
        const cudaGraphNode_t* deps = nullptr;
        size_t ndeps = 0;
        e = cudaStreamGetCaptureInfo(h->stream, &st, nullptr, nullptr, &deps, &ndeps);
        std::vector<cudaGraphNode_t> tails(deps, deps + (e == cudaSuccess ? ndeps : 0));
        cudaError_t e2 = cudaStreamEndCapture(h->stream, &dummy);
        if (e != cudaSuccess || e2 != cudaSuccess) return fail(e != cudaSuccess ? e : e2);
        h->loop_launches_head[gi] = count;
        // WHILE node and its body
        cudaGraphNodeParams np = {};
        np.type = cudaGraphNodeTypeConditional;
        np.conditional.handle = handle;
        np.conditional.type = cudaGraphCondTypeWhile;
        np.conditional.size = 1;
        cudaGraphNode_t wnode;
        if ((e = cudaGraphAddNode(&wnode, g, tails.data(), tails.size(), &np)) != cudaSuccess) return fail(e);
        cudaGraph_t body = np.conditional.phGraph_out[0];
        count = 0;
        if ((e = cudaStreamBeginCaptureToGraph(h->stream, body, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed)) != cudaSuccess) return fail(e);
        enqueue_loop_body(h, handle, norm_out, &count);
        if ((e = cudaStreamEndCapture(h->stream, &dummy)) != cudaSuccess) return fail(e);
        h->loop_launches_body[gi] = count;
        if ((e = cudaGraphInstantiate(&h->loop_exec[gi], g, 0)) != cudaSuccess) return fail(e);
        h->loop_epoch[gi] = h->graph_epoch;
    }
    const int max = (int)h->h_loop[2];
    cudaError_t e = cudaMemcpyAsync(h->d_loop, h->h_loop, 9 * sizeof(double), cudaMemcpyHostToDevice, h->stream);
    if (e == cudaSuccess) e = cudaGraphLaunch(h->loop_exec[gi], h->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(h->h_loop, h->d_loop, (size_t)(8 + max + 1) * sizeof(double), cudaMemcpyDeviceToHost, h->stream);
    if (e != cudaSuccess) return fail(e);
    return VMG_OK;
}

// ------------------------------------------------------------------------------------------------
// N1, kernel level: the coarser levels (segment 1 of the cycle) of ALL members of a vmg_create_batch group as one graph
// whose launches run over planes x problems (LevelView::pstride), K CTAs in the tail.  Level 0 stays one problem at a
// time (segments 0 and 2 of each member), which keeps the L2 reuse between its consecutive half-sweeps.
// ------------------------------------------------------------------------------------------------
inline bool group_coarse_ok(const VmgBatchGroup* G)
{
    const vmg_s* a = G->members[0];
    if (!vcycle_segmentable(a) || a->use_blocked || a->prolong || a->nu2 < 1) return false;
    for (const vmg_s* h : G->members) {
        if (!h->have_coeffs || !h->have_bc || !vcycle_segmentable(h)) return false;
        if (h->nu1 != a->nu1 || h->nu2 != a->nu2 || h->nbottom != a->nbottom || h->prolong != a->prolong || h->symmetric != a->symmetric ||
            h->use_tail != a->use_tail || h->tail_level != a->tail_level || h->use_pdl != a->use_pdl || h->snake != a->snake ||
            h->use_blocked != a->use_blocked)
            return false;
        for (int l = 1; l < h->nlev; ++l) {
            const VmgLevel &x = h->lev[l], &y = a->lev[l];
            if (x.cw != y.cw || (x.cw && (x.cx != y.cx || x.cy != y.cy || x.cz != y.cz))) return false;   // constant weights go by value
        }
    }
    return true;
}

// every level of ALL members in one graph (all problems still iterating and K level-0 working sets small enough to share
// the L2): the whole V-cycle + the K residual norms as problem-major launches
inline bool group_full_ok(const VmgBatchGroup* G)
{
    const vmg_s* a = G->members[0];
    const long long K = (long long)G->members.size();
    if ((double)K * a->lev[0].n * 56.0 > a->batch_full_mb * 1048576.0 || (long long)a->lev[0].nz * K * 2 > 65535) return false;
    for (const vmg_s* h : G->members) {
        const VmgLevel &x = h->lev[0], &y = a->lev[0];
        if (h->d_mask || x.cw != y.cw || (x.cw && (x.cx != y.cx || x.cy != y.cy || x.cz != y.cz))) return false;
    }
    return true;
}

inline int run_group_full(VmgBatchGroup* G)
{
    vmg_s* h = G->members[0];
    const int K = (int)G->members.size();
    bool stale = G->full_exec == nullptr;
    for (int i = 0; i < K; ++i) stale = stale || G->full_epochs[i] != G->members[i]->graph_epoch;
    if (stale) {
        if (G->full_exec) { cudaGraphExecDestroy(G->full_exec); G->full_exec = nullptr; }
        if (G->full_graph) { cudaGraphDestroy(G->full_graph); G->full_graph = nullptr; }
        const long long stride = (long long)(G->stride_bytes / sizeof(double));
        for (int l = 0; l < h->nlev; ++l) { h->lev[l].nprob = K; h->lev[l].pstride = stride; }
        long long count = 0;
        unsigned long long* out0 = (unsigned long long*)h->d_scal + 1;
        cudaError_t e = cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeRelaxed);
        if (e == cudaSuccess) {
            for (int i = 1; i < K; ++i) cudaMemsetAsync(out0 + (long long)i * stride, 0, sizeof(unsigned long long), h->stream);
            enqueue_vcycle(h, out0, &count);
            e = cudaStreamEndCapture(h->stream, &G->full_graph);
        }
        for (int l = 0; l < h->nlev; ++l) { h->lev[l].nprob = 1; h->lev[l].pstride = 0; }
        if (e == cudaSuccess) e = cudaGraphInstantiate(&G->full_exec, G->full_graph, 0);
        if (e != cudaSuccess) { h->last_cuda_error = (int)e; (void)cudaGetLastError(); return VMG_ERR_CUDA; }
        G->full_launches = count;
        for (int i = 0; i < K; ++i) G->full_epochs[i] = G->members[i]->graph_epoch;
    }
    cudaError_t e = cudaGraphLaunch(G->full_exec, h->stream);
    if (e != cudaSuccess) { h->last_cuda_error = (int)e; (void)cudaGetLastError(); return VMG_ERR_CUDA; }
    return VMG_OK;
}

inline int run_group_coarse(VmgBatchGroup* G)
{
    vmg_s* h = G->members[0];
    bool stale = G->coarse_exec == nullptr;
    for (size_t i = 0; i < G->members.size(); ++i) stale = stale || G->coarse_epochs[i] != G->members[i]->graph_epoch;
    if (stale) {
        if (G->coarse_exec) { cudaGraphExecDestroy(G->coarse_exec); G->coarse_exec = nullptr; }
        if (G->coarse_graph) { cudaGraphDestroy(G->coarse_graph); G->coarse_graph = nullptr; }
        const int K = (int)G->members.size();
        for (int l = 0; l < h->nlev; ++l) h->lev[l].cur = 0;
        for (int l = 1; l < h->nlev; ++l) { h->lev[l].nprob = K; h->lev[l].pstride = (long long)(G->stride_bytes / sizeof(double)); }
        long long count = 0;
        cudaError_t e = cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeRelaxed);
        if (e == cudaSuccess) {
            enqueue_vcycle_segment(h, 1, nullptr, &count);
            e = cudaStreamEndCapture(h->stream, &G->coarse_graph);
        }
        for (int l = 1; l < h->nlev; ++l) { h->lev[l].nprob = 1; h->lev[l].pstride = 0; }
        if (e == cudaSuccess) e = cudaGraphInstantiate(&G->coarse_exec, G->coarse_graph, 0);
        if (e != cudaSuccess) { h->last_cuda_error = (int)e; (void)cudaGetLastError(); return VMG_ERR_CUDA; }
        G->coarse_launches = count;
        for (size_t i = 0; i < G->members.size(); ++i) G->coarse_epochs[i] = G->members[i]->graph_epoch;
    }
    cudaError_t e = cudaGraphLaunch(G->coarse_exec, h->stream);
    if (e != cudaSuccess) { h->last_cuda_error = (int)e; (void)cudaGetLastError(); return VMG_ERR_CUDA; }
    return VMG_OK;
}

// V-cycle followed by the residual norm into *out (device), as a graph replay when enabled.
inline int run_vcycle_with_norm(vmg_s* h, unsigned long long* out)
{
    prepare_blocked(h);
    auto body = [&](long long* count) { enqueue_vcycle(h, out, count); };
    if (!h->use_graph || h->profile) {
        long long count = 0;
        body(&count);
        h->launches += count;
        h->launches_per_cycle = count;
        if (cudaGetLastError() != cudaSuccess) return VMG_ERR_CUDA;
        return VMG_OK;
    }
    const int gi = h->lev[0].cw;
    if (h->graph_slot_epoch[gi] != h->graph_epoch) {
        own_l2_window(h);
        if (h->graph_exec[gi]) { cudaGraphExecDestroy(h->graph_exec[gi]); h->graph_exec[gi] = nullptr; }
        if (h->graph[gi]) { cudaGraphDestroy(h->graph[gi]); h->graph[gi] = nullptr; }
        long long count = 0;
        if (cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeRelaxed) != cudaSuccess) {
            h->last_cuda_error = (int)cudaGetLastError();
            return VMG_ERR_CUDA;
        }
        body(&count);
        cudaError_t e = cudaStreamEndCapture(h->stream, &h->graph[gi]);
        if (e == cudaSuccess) e = cudaGraphInstantiate(&h->graph_exec[gi], h->graph[gi], 0);
        if (e != cudaSuccess) { h->last_cuda_error = (int)e; (void)cudaGetLastError(); return VMG_ERR_CUDA; }
        h->graph_slot_launches[gi] = count;
        h->graph_slot_epoch[gi] = h->graph_epoch;
    }
    h->launches_per_cycle = h->graph_slot_launches[gi];
    cudaError_t e = cudaGraphLaunch(h->graph_exec[gi], h->stream);
    if (e != cudaSuccess) { h->last_cuda_error = (int)e; (void)cudaGetLastError(); return VMG_ERR_CUDA; }
    h->launches += h->launches_per_cycle;
    return VMG_OK;
}

}  // namespace vmg
