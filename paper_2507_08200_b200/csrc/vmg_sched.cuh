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
            smooth_colour_kernel<<<grid_for(nt), kThreads, 0, h->stream>>>(v, phi, rhs, colour);
            ++*count;
        }
}

inline void enqueue_residual_restrict(vmg_s* h, int l, const double* phi, const double* rhs, double* crhs,
                                      double* cphi, long long* count)
{
    VmgLevel& L = h->lev[l];
    ProfScope ps(h, l == 0 ? VMG_PC_RESREST0 : VMG_PC_COARSE, count);
    residual_restrict_kernel<<<grid_for(h->lev[l + 1].n), kThreads, 0, h->stream>>>(view(L), phi, rhs, crhs, cphi,
                                                                                    h->three_d ? 2 : 1);
    ++*count;
}

inline void enqueue_prolong_correct(vmg_s* h, int l, double* phi, const double* e, long long* count)
{
    VmgLevel& L = h->lev[l];
    ProfScope ps(h, l == 0 ? VMG_PC_PROLONG0 : VMG_PC_COARSE, count);
    prolong_correct_kernel<<<grid_for(L.n), kThreads, 0, h->stream>>>(phi, e, L.nx, L.ny, L.nz, h->three_d ? 2 : 1);
    ++*count;
}

inline void enqueue_residual_norm(vmg_s* h, unsigned long long* out)
{
    VmgLevel& L = h->lev[0];
    unsigned g = std::min<unsigned>(grid_for(L.n), 8u * (unsigned)h->num_sms);
    ProfScope ps(h, VMG_PC_NORM, nullptr);
    residual_norm_kernel<<<g, kThreads, 0, h->stream>>>(view(L), L.phi, L.rhs, out);
}

// C4: one V-cycle on the handle's own level arrays (level-0 phi / rhs = btilde already in place).
inline void enqueue_vcycle(vmg_s* h, long long* count)
{
    int last = h->nlev - 1;
    for (int l = 0; l < last; ++l) {
        VmgLevel& L = h->lev[l];
        enqueue_smooth(h, l, L.phi, L.rhs, h->nu1, count);
        enqueue_residual_restrict(h, l, L.phi, L.rhs, h->lev[l + 1].rhs, h->lev[l + 1].phi, count);
    }
    {
        VmgLevel& B = h->lev[last];
        if (last == 0) cudaMemsetAsync(B.phi, 0, B.n * sizeof(double), h->stream);   // single level: bottom from zero
        enqueue_smooth(h, last, B.phi, B.rhs, h->nbottom, count);
    }
    for (int l = last - 1; l >= 0; --l) {
        VmgLevel& L = h->lev[l];
        enqueue_prolong_correct(h, l, L.phi, h->lev[l + 1].phi, count);
        enqueue_smooth(h, l, L.phi, L.rhs, h->nu2, count);
    }
}

// V-cycle followed by the residual norm into *out (device), as a graph replay when enabled.
inline int run_vcycle_with_norm(vmg_s* h, unsigned long long* out)
{
    auto body = [&](long long* count) {
        enqueue_vcycle(h, count);
        cudaMemsetAsync(out, 0, sizeof(unsigned long long), h->stream);
        enqueue_residual_norm(h, out);
        ++*count;
    };
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
        if (cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
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
