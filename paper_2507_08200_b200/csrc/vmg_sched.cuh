// vmg_sched.cuh -- sequencing of one V-cycle (S7): which kernel runs each step on each level, plain
// launches or one CUDA graph replay (north_star (4)).
#pragma once
#include "vmg_internal.h"
#include "vmg_kernels.cuh"
#include "../../include/vmg.h"
#include <algorithm>

namespace vmg {

inline LevelView view(const VmgLevel& L)
{
    LevelView v;
    v.wx = L.wx; v.wy = L.wy; v.wz = L.wz; v.dinv = L.dinv;
    v.nx = L.nx; v.ny = L.ny; v.nz = L.nz; v.nxy = (long long)L.nx * L.ny; v.n = L.n;
    return v;
}

inline unsigned grid_for(long long n) { return (unsigned)cdiv(n, kThreads); }

inline void plan_schedule(vmg_s* h) { (void)h; }

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

inline int enqueue_fold_bc(vmg_s* h, const double* rhs, double* bt)
{
    VmgLevel& L = h->lev[0];
    FoldArgs g;
    g.rhs = rhs; g.bt = bt;
    for (int f = 0; f < 6; ++f) {
        g.wb[f] = L.wb[f];
        g.val[f] = h->bc_has_value[f] ? h->bcval[f] : nullptr;
        g.dirichlet[f] = h->bctype[f] == VMG_BC_DIRICHLET;
    }
    g.nx = L.nx; g.ny = L.ny; g.nz = L.nz; g.three_d = h->three_d;
    g.h[0] = L.hx; g.h[1] = L.hy; g.h[2] = L.hz;
    {
        ProfScope ps(h, VMG_PC_FOLD, nullptr);
        fold_bc_kernel<<<grid_for(L.n), kThreads, 0, h->stream>>>(g);
    }
    h->launches += 1;
    return cudaGetLastError() == cudaSuccess ? VMG_OK : VMG_ERR_CUDA;
}

// counts launches into *count
inline void enqueue_smooth(vmg_s* h, int l, double* phi, const double* rhs, int nsweeps, long long* count)
{
    VmgLevel& L = h->lev[l];
    LevelView v = view(L);
    ProfScope ps(h, l == 0 ? VMG_PC_SMOOTH0 : VMG_PC_COARSE, count);
    long long nt = (long long)((L.nx + 1) / 2) * L.ny * L.nz;
    for (int s = 0; s < nsweeps; ++s)
        for (int colour = 0; colour < 2; ++colour) {
            smooth_colour_kernel<<<grid_for(nt), kThreads, 0, h->stream>>>(v, phi, rhs, colour, 0, L.nz);
            ++*count;
        }
}

inline void enqueue_residual_restrict(vmg_s* h, int l, const double* phi, const double* rhs, double* crhs,
                                      double* cphi, long long* count)
{
    VmgLevel& L = h->lev[l];
    ProfScope ps(h, l == 0 ? VMG_PC_RESREST0 : VMG_PC_COARSE, count);
    residual_restrict_kernel<<<grid_for(h->lev[l + 1].n), kThreads, 0, h->stream>>>(view(L), phi, rhs, crhs, cphi,
                                                                                    h->three_d ? 2 : 1, 0, h->lev[l + 1].nz);
    ++*count;
}

inline void enqueue_prolong_correct(vmg_s* h, int l, double* phi, const double* e, long long* count)
{
    VmgLevel& L = h->lev[l];
    ProfScope ps(h, l == 0 ? VMG_PC_PROLONG0 : VMG_PC_COARSE, count);
    prolong_correct_kernel<<<grid_for(L.n), kThreads, 0, h->stream>>>(phi, e, L.nx, L.ny, h->three_d ? 2 : 1, 0, L.nz);
    ++*count;
}

inline void enqueue_residual_norm(vmg_s* h, unsigned long long* out)
{
    VmgLevel& L = h->lev[0];
    unsigned g = std::min<unsigned>(grid_for(L.n), 8u * (unsigned)h->num_sms);
    ProfScope ps(h, VMG_PC_NORM, nullptr);
    residual_norm_kernel<<<g, kThreads, 0, h->stream>>>(view(L), L.phi, L.rhs, out, 0, L.nz);
}

// ------------------------------------------------------------------------------------------------
// L2 wavefront schedule for one stroke of a level.  A stroke is a list of stages, each a
// whole-level operation whose value at plane k depends on the previous stage at planes k-1, k, k+1 only:
//   down-stroke: red, black (x nu1), residual+restriction          up-stroke: prolongation+correction, red, black (x nu2)
//   [, residual norm].  Stage s of slab j covers planes [j*T - s, (j+1)*T - s): a parallelogram tiling of (z, stage)
// without redundant work.  Stage s runs on its own stream, in slab order; it waits for stage s-1 of the same slab.
// Up to S launches on S consecutive slabs are in flight together and the slabs they touch (about (S+1)*T planes of
// the six arrays) stay resident in the 126 MB L2, so HBM sees each array once per stroke instead of once per stage.
// Under stream capture the cross-stream events become edges of the V-cycle's CUDA graph.
// ------------------------------------------------------------------------------------------------
enum StageKind { ST_SMOOTH = 0, ST_RESREST = 1, ST_PROLONG = 2, ST_NORM = 3 };
struct Stage { int kind; int colour; };

inline bool use_wavefront(const vmg_s* h, int l)
{
    const VmgLevel& L = h->lev[l];
    return h->use_blocked && h->wf_planes >= 2 && h->three_d && L.n >= h->wf_min_cells && L.nz >= 4 * h->wf_planes &&
           l + 1 < h->nlev;
}

inline void launch_stage(vmg_s* h, int l, const Stage& st, int k0, int k1, cudaStream_t stream, unsigned long long* norm_out)
{
    VmgLevel& L = h->lev[l];
    LevelView v = view(L);
    int sz = h->three_d ? 2 : 1;
    switch (st.kind) {
    case ST_SMOOTH: {
        long long nt = (long long)((L.nx + 1) / 2) * L.ny * (k1 - k0);
        smooth_colour_kernel<<<grid_for(nt), kThreads, 0, stream>>>(v, L.phi, L.rhs, st.colour, k0, k1);
        break;
    }
    case ST_RESREST: {
        VmgLevel& C = h->lev[l + 1];
        long long nt = (long long)C.nx * C.ny * ((k1 - k0) / 2);
        residual_restrict_kernel<<<grid_for(nt), kThreads, 0, stream>>>(v, L.phi, L.rhs, C.rhs, C.phi, sz, k0 / 2, k1 / 2);
        break;
    }
    case ST_PROLONG: {
        long long nt = (long long)L.nx * L.ny * (k1 - k0);
        prolong_correct_kernel<<<grid_for(nt), kThreads, 0, stream>>>(L.phi, h->lev[l + 1].phi, L.nx, L.ny, sz, k0, k1);
        break;
    }
    case ST_NORM: {
        long long nt = (long long)L.nx * L.ny * (k1 - k0);
        unsigned g = std::min<unsigned>(grid_for(nt), 8u * (unsigned)h->num_sms);
        residual_norm_kernel<<<g, kThreads, 0, stream>>>(v, L.phi, L.rhs, norm_out, k0, k1);
        break;
    }
    }
}

// creates the side streams and the event pool (outside any stream capture)
inline void prepare_wavefront(vmg_s* h)
{
    size_t need = 0;
    for (int l = 0; l + 1 < h->nlev; ++l)
        if (use_wavefront(h, l)) {
            size_t S = 2 * (size_t)std::max(h->nu1, h->nu2) + 2;
            size_t J = (size_t)cdiv(h->lev[l].nz + (long long)S - 1, h->wf_planes);
            need = std::max(need, S * J + S + 1);
        }
    if (need == 0) return;
    if (!h->side_ready) {
        for (int s = 0; s < vmg_s::kMaxStages; ++s) cudaStreamCreateWithFlags(&h->side[s], cudaStreamNonBlocking);
        h->side_ready = true;
    }
    while (h->wf_events.size() < need) {
        cudaEvent_t e;
        cudaEventCreateWithFlags(&e, cudaEventDisableTiming);
        h->wf_events.push_back(e);
    }
}

inline void enqueue_wavefront(vmg_s* h, int l, const std::vector<Stage>& stages, unsigned long long* norm_out, long long* count)
{
    VmgLevel& L = h->lev[l];
    const int S = (int)stages.size(), T = h->wf_planes, nz = L.nz;
    const int J = (int)cdiv(nz + S - 1, T);
    if ((size_t)S * J + S + 1 > h->wf_events.size()) return;   // prepare_wavefront() sizes the pool; cannot happen
    auto ev = [&](int s, int j) { return h->wf_events[(size_t)s * J + j]; };
    cudaEvent_t fork = h->wf_events[(size_t)S * J + S];
    cudaEventRecord(fork, h->stream);
    for (int s = 0; s < S; ++s) cudaStreamWaitEvent(h->side[s], fork, 0);
    for (int j = 0; j < J; ++j)
        for (int s = 0; s < S; ++s) {
            int k0 = std::max(0, j * T - s), k1 = std::min(nz, (j + 1) * T - s);
            if (s > 0) cudaStreamWaitEvent(h->side[s], ev(s - 1, j), 0);
            if (k1 > k0) { launch_stage(h, l, stages[s], k0, k1, h->side[s], norm_out); ++*count; }
            cudaEventRecord(ev(s, j), h->side[s]);
        }
    for (int s = 0; s < S; ++s) {
        cudaEvent_t done = h->wf_events[(size_t)S * J + s];
        cudaEventRecord(done, h->side[s]);
        cudaStreamWaitEvent(h->stream, done, 0);
    }
}

// down-stroke of level l: nu1 sweeps then residual+restriction into level l+1 (which also zeroes its phi)
inline void enqueue_down(vmg_s* h, int l, long long* count)
{
    VmgLevel& L = h->lev[l];
    if (use_wavefront(h, l) && (h->wf_planes % 2 == 0)) {
        ProfScope ps(h, l == 0 ? VMG_PC_SMOOTH0 : VMG_PC_COARSE, count);
        std::vector<Stage> st;
        for (int s = 0; s < h->nu1; ++s) { st.push_back({ST_SMOOTH, 0}); st.push_back({ST_SMOOTH, 1}); }
        st.push_back({ST_RESREST, 0});
        enqueue_wavefront(h, l, st, nullptr, count);
        return;
    }
    enqueue_smooth(h, l, L.phi, L.rhs, h->nu1, count);
    enqueue_residual_restrict(h, l, L.phi, L.rhs, h->lev[l + 1].rhs, h->lev[l + 1].phi, count);
}

// up-stroke of level l: prolongation+correction from level l+1 then nu2 sweeps [then the residual norm (level 0)]
// returns true if the residual norm was fused into the stroke
inline bool enqueue_up(vmg_s* h, int l, unsigned long long* norm_out, long long* count)
{
    VmgLevel& L = h->lev[l];
    if (use_wavefront(h, l)) {
        ProfScope ps(h, l == 0 ? VMG_PC_SMOOTH0 : VMG_PC_COARSE, count);
        std::vector<Stage> st;
        st.push_back({ST_PROLONG, 0});
        for (int s = 0; s < h->nu2; ++s) { st.push_back({ST_SMOOTH, 0}); st.push_back({ST_SMOOTH, 1}); }
        bool fuse_norm = (l == 0 && norm_out != nullptr);
        if (fuse_norm) st.push_back({ST_NORM, 0});
        enqueue_wavefront(h, l, st, norm_out, count);
        return fuse_norm;
    }
    enqueue_prolong_correct(h, l, L.phi, h->lev[l + 1].phi, count);
    enqueue_smooth(h, l, L.phi, L.rhs, h->nu2, count);
    return false;
}

// C4: one V-cycle on the handle's own level arrays (level-0 phi / rhs = btilde already in place).
// If norm_out is given, *norm_out (zeroed here) receives the bit pattern of ||rhs - A phi||_inf on level 0.
inline void enqueue_vcycle(vmg_s* h, unsigned long long* norm_out, long long* count)
{
    int last = h->nlev - 1;
    if (norm_out) cudaMemsetAsync(norm_out, 0, sizeof(unsigned long long), h->stream);
    for (int l = 0; l < last; ++l) enqueue_down(h, l, count);
    {
        VmgLevel& B = h->lev[last];
        if (last == 0) cudaMemsetAsync(B.phi, 0, B.n * sizeof(double), h->stream);   // single level: bottom from zero
        enqueue_smooth(h, last, B.phi, B.rhs, h->nbottom, count);
    }
    bool norm_done = false;
    for (int l = last - 1; l >= 0; --l) norm_done = enqueue_up(h, l, l == 0 ? norm_out : nullptr, count);
    if (norm_out && !norm_done) { enqueue_residual_norm(h, norm_out); ++*count; }
}

// V-cycle followed by the residual norm into *out (device), as a graph replay when enabled.
inline int run_vcycle_with_norm(vmg_s* h, unsigned long long* out)
{
    prepare_wavefront(h);
    auto body = [&](long long* count) { enqueue_vcycle(h, out, count); };
    if (!h->use_graph || h->profile) {
        long long count = 0;
        body(&count);
        h->launches += count;
        h->launches_per_cycle = count;
        if (cudaGetLastError() != cudaSuccess) return VMG_ERR_CUDA;
        return VMG_OK;
    }
    if (!h->graph_valid) {
        if (h->graph_exec) { cudaGraphExecDestroy(h->graph_exec); h->graph_exec = nullptr; }
        if (h->graph) { cudaGraphDestroy(h->graph); h->graph = nullptr; }
        long long count = 0;
        if (cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeRelaxed) != cudaSuccess) {
            h->last_cuda_error = (int)cudaGetLastError();
            return VMG_ERR_CUDA;
        }
        body(&count);
        cudaError_t e = cudaStreamEndCapture(h->stream, &h->graph);
        if (e == cudaSuccess) e = cudaGraphInstantiate(&h->graph_exec, h->graph, 0);
        if (e != cudaSuccess) { h->last_cuda_error = (int)e; (void)cudaGetLastError(); return VMG_ERR_CUDA; }
        h->launches_per_cycle = count;
        h->graph_valid = true;
    }
    cudaError_t e = cudaGraphLaunch(h->graph_exec, h->stream);
    if (e != cudaSuccess) { h->last_cuda_error = (int)e; (void)cudaGetLastError(); return VMG_ERR_CUDA; }
    h->launches += h->launches_per_cycle;
    return VMG_OK;
}

}  // namespace vmg
