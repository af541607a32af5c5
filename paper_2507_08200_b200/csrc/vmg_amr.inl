// vmg_amr.inl -- C-ABI of the two-level composite solve (include/vmg.h, "vmg_amr_*"; kernels and the design in
// vmg_amr.cuh).  Included at the end of vmg_api.cu: it uses the single-level handles' internals.

#include "vmg_amr.cuh"

struct vmg_amr_s {
    vmg_s* hc = nullptr;            // the coarse box (an ordinary handle: correction V-cycle, fold_bc)
    std::vector<vmg_s*> hf;         // the patches (ordinary handles whose faces are coarse-fine faces)
    std::vector<AmrGeom> A;         // per patch: box, patch and shadow geometry
    cudaStream_t stream = nullptr;
    // several patches: every patch handle runs on a stream of its own, forked from and joined to `stream` around each per-patch
    // section (amr_fork / amr_join) -- inside the captured graphs the patches are parallel branches (their kernels are small
    // and latency-bound: one patch of 128 x 64 x 64 cells fills the GPU once).  One patch: it shares `stream`.
    std::vector<cudaStream_t> ps;
    cudaEvent_t ev_fork = nullptr;
    std::vector<cudaEvent_t> ev_join;
    void* base = nullptr;           // one allocation: btilde_c (padded like a level array), per patch rhs_f copy and shadow means, scalars
    double* btc = nullptr;
    std::vector<double*> rhsf, old;
    unsigned long long* d_norm = nullptr;   // ||btilde_c||, ||f_f||, ||r_c||, ||r_f|| (bit patterns; the fine ones over all patches)
    double* h_norm = nullptr;       // pinned mirror
    int nu_f = 6;                   // A4: fine sweeps per cycle
    bool have_coeffs = false, have_bc = false;
    cudaGraph_t graph[3] = {nullptr, nullptr, nullptr};   // 0: composite residual + norms (every cell), 1: correction + fine sweeps,
    cudaGraphExec_t exec[3] = {nullptr, nullptr, nullptr};   // 2: as 0 with the coarse norm over the red cells (after a V-cycle, R12)
    long long graph_launches[3] = {0, 0, 0};
    // the cycle loop as ONE graph with a conditional WHILE node (as vmg_solve): body = correction + composite
    // residual + solve_decide_kernel; used when the coarse handle's options allow it (device_loop, graph, no profile)
    cudaGraph_t loop_graph = nullptr;
    cudaGraphExec_t loop_exec = nullptr;
    long long loop_launches = 0;
    double *d_loop = nullptr, *h_loop = nullptr;   // nb, rtol, max, cycles, slow, status, -, -, hist[kLoopMaxCycles + 1] (device / pinned)
    unsigned epoch_c = 0;
    std::vector<unsigned> epoch_f;
    int graph_nu_f = -1;
    int cycles = 0, last_cuda_error = 0;
    double relres = 0.0;
    std::vector<double> hist;
    long long launches = 0;
    int np() const { return (int)hf.size(); }
};

#define AMR_TRY(A_, expr)                                                      \
    do {                                                                       \
        cudaError_t e__ = (expr);                                              \
        if (e__ != cudaSuccess) {                                              \
            (A_)->last_cuda_error = (int)e__;                                  \
            (void)cudaGetLastError();                                          \
            return VMG_ERR_CUDA;                                               \
        }                                                                      \
    } while (0)

namespace {

cudaStream_t amr_pstream(const vmg_amr_s* a, int q) { return a->ps.empty() ? a->stream : a->ps[q]; }

void amr_fork(vmg_amr_s* a)
{
    if (a->ps.empty()) return;
    cudaEventRecord(a->ev_fork, a->stream);
    for (cudaStream_t s : a->ps) cudaStreamWaitEvent(s, a->ev_fork, 0);
}

void amr_join(vmg_amr_s* a)
{
    for (size_t q = 0; q < a->ps.size(); ++q) {
        cudaEventRecord(a->ev_join[q], a->ps[q]);
        cudaStreamWaitEvent(a->stream, a->ev_join[q], 0);
    }
}

void amr_drop_graphs(vmg_amr_s* a)
{
    for (int i = 0; i < 3; ++i) {
        if (a->exec[i]) { cudaGraphExecDestroy(a->exec[i]); a->exec[i] = nullptr; }
        if (a->graph[i]) { cudaGraphDestroy(a->graph[i]); a->graph[i] = nullptr; }
    }
    if (a->loop_exec) { cudaGraphExecDestroy(a->loop_exec); a->loop_exec = nullptr; }
    if (a->loop_graph) { cudaGraphDestroy(a->loop_graph); a->loop_graph = nullptr; }
}

// value planes of patch q from the coarse field, then btilde_f = f_f + 2 wb g (the library's fold_bc)
int amr_enqueue_ghost_fold(vmg_amr_s* a, int q, long long* count)
{
    vmg_s* hf = a->hf[q];
    AmrGhostArgs g;
    g.A = a->A[q]; g.phic = a->hc->lev[0].phi;
    long long most = 0;
    for (int f = 0; f < 6; ++f) {
        g.plane[f] = hf->bcval[f];
        if (f < 2 * g.A.nd) most = std::max<long long>(most, (long long)plane_count(hf->lev[0], f));
    }
    amr_ghost_kernel<<<dim3(grid_for(most), 2 * g.A.nd), kThreads, 0, amr_pstream(a, q)>>>(g);
    ++*count;
    long long before = hf->launches;
    int rc = enqueue_fold_bc(hf, a->rhsf[q], hf->lev[0].rhs);
    *count += hf->launches - before;
    return rc;
}

// graphs 0 / 2: the composite residual (A3) -- every patch's residual + restriction and residual norm, the coarse right-hand
// side in and next to every patch, then the library's residual norm of the box on that right-hand side (amr_patch_rhs_kernel)
void amr_enqueue_residual(vmg_amr_s* a, long long* count, bool red_only)
{
    vmg_s* hc = a->hc;
    cudaMemsetAsync(a->d_norm + 2, 0, sizeof(unsigned long long), a->stream);   // the maximum of A5 over both levels: one scalar
    amr_fork(a);
    for (int q = 0; q < a->np(); ++q) {
        vmg_s* hf = a->hf[q];
        hf->lev[0].cur = 0;
        plain_residual_restrict(hf, 0, count);
        enqueue_residual_norm(hf, a->d_norm + 2);
        ++*count;
        AmrResArgs g;
        g.A = a->A[q]; g.Lc = view(hc->lev[0]);
        g.phic = hc->lev[0].phi; g.btc = a->btc; g.rs = hf->lev[1].rhs; g.phif = hf->lev[0].phi;
        g.R = hc->lev[0].rhs;
        for (int f = 0; f < 6; ++f) { g.gplane[f] = hf->bcval[f]; g.wbf[f] = hf->lev[0].wb[f]; }
        g.wscale = 2.0 / (double)(1 << g.A.nd);
        g.norm = a->d_norm + 2;
        long long region = 1;
        for (int d = 0; d < g.A.nd; ++d) region *= g.A.hi[d] - g.A.lo[d] + 2;
        amr_patch_rhs_kernel<<<grid_for(region), kThreads, 0, amr_pstream(a, q)>>>(g);
        ++*count;
    }
    amr_join(a);
    hc->lev[0].cur = 0;
    enqueue_residual_norm(hc, a->d_norm + 2, red_only);
    ++*count;
}

// graph 1: A4 after the exit test -- coarse V-cycle (in place on phi_c, right-hand side of amr_patch_rhs_kernel), then per
// patch: correction, ghosts, fine sweeps, average down
int amr_enqueue_correction(vmg_amr_s* a, long long* count)
{
    vmg_s* hc = a->hc;
    VmgLevel& C0 = hc->lev[0];
    enqueue_vcycle(hc, nullptr, count);
    amr_fork(a);
    int rc_all = VMG_OK;
    for (int q = 0; q < a->np(); ++q) {
        vmg_s* hf = a->hf[q];
        const AmrGeom& A = a->A[q];
        cudaStream_t sq = amr_pstream(a, q);
        amr_prolong_add_kernel<<<grid_for(A.F.n), kThreads, 0, sq>>>(A, hf->lev[0].phi, C0.phi, a->old[q]);
        ++*count;
        int rc = amr_enqueue_ghost_fold(a, q, count);
        if (rc != VMG_OK) rc_all = rc;           // keep going: the forked streams have to be joined before a capture can end
        hf->lev[0].cur = 0; hf->lev[0].dir = 0;
        plain_smooth(hf, 0, a->nu_f, count);
        amr_average_down_kernel<<<grid_for(A.S.n), kThreads, 0, sq>>>(A, hf->lev[0].phi, C0.phi, a->old[q]);
        ++*count;
    }
    amr_join(a);
    return rc_all;
}

bool amr_graphs_current(const vmg_amr_s* a)
{
    if (!a->exec[0] || a->epoch_c != a->hc->graph_epoch || a->graph_nu_f != a->nu_f) return false;
    for (int q = 0; q < a->np(); ++q) if (a->epoch_f[q] != a->hf[q]->graph_epoch) return false;
    return true;
}

// runs part `which` (0 residual over every cell, 1 correction, 2 residual with the coarse norm over the red cells): a graph
// replay, or plain launches with option graph = 0 / profile on the coarse handle
int amr_run(vmg_amr_s* a, int which)
{
    vmg_s* hc = a->hc;
    if (!hc->use_graph || hc->profile) {
        long long count = 0;
        int rc = VMG_OK;
        if (which != 1) amr_enqueue_residual(a, &count, which == 2); else rc = amr_enqueue_correction(a, &count);
        a->launches += count;
        if (rc != VMG_OK) return rc;
        AMR_TRY(a, cudaGetLastError());
        return VMG_OK;
    }
    if (!amr_graphs_current(a)) {
        amr_drop_graphs(a);
        for (int i = 0; i < 3; ++i) {
            long long count = 0;
            AMR_TRY(a, cudaStreamBeginCapture(a->stream, cudaStreamCaptureModeRelaxed));
            int rc = VMG_OK;
            if (i != 1) amr_enqueue_residual(a, &count, i == 2); else rc = amr_enqueue_correction(a, &count);
            cudaError_t e = cudaStreamEndCapture(a->stream, &a->graph[i]);
            if (rc != VMG_OK) return rc;
            if (e == cudaSuccess) e = cudaGraphInstantiate(&a->exec[i], a->graph[i], 0);
            AMR_TRY(a, e);
            a->graph_launches[i] = count;
        }
        a->epoch_c = hc->graph_epoch; a->graph_nu_f = a->nu_f;
        for (int q = 0; q < a->np(); ++q) a->epoch_f[q] = a->hf[q]->graph_epoch;
    }
    if (which < 0) return VMG_OK;            // only (re)capture
    AMR_TRY(a, cudaGraphLaunch(a->exec[which], a->stream));
    a->launches += a->graph_launches[which];
    return VMG_OK;
}

// The cycles after the first residual as one graph launch: WHILE (continue) { correction; composite residual (coarse norm over
// the red cells); solve_decide_kernel: history, exit rules C5, sets `continue` }.  The caller has filled h_loop[0..8] and hist[0].
int amr_run_loop(vmg_amr_s* a)
{
    if (!a->loop_exec || !amr_graphs_current(a)) {
        if (a->loop_exec) { cudaGraphExecDestroy(a->loop_exec); a->loop_exec = nullptr; }
        if (a->loop_graph) { cudaGraphDestroy(a->loop_graph); a->loop_graph = nullptr; }
        cudaGraph_t g = nullptr, dummy = nullptr;
        AMR_TRY(a, cudaGraphCreate(&g, 0));
        a->loop_graph = g;
        cudaGraphConditionalHandle handle;
        AMR_TRY(a, cudaGraphConditionalHandleCreate(&handle, g, 1, cudaGraphCondAssignDefault));
        cudaGraphNodeParams np = {};
        np.type = cudaGraphNodeTypeConditional;
        np.conditional.handle = handle;
        np.conditional.type = cudaGraphCondTypeWhile;
        np.conditional.size = 1;
        cudaGraphNode_t wnode;
        AMR_TRY(a, cudaGraphAddNode(&wnode, g, nullptr, 0, &np));
        cudaGraph_t body = np.conditional.phGraph_out[0];
        long long count = 0;
        AMR_TRY(a, cudaStreamBeginCaptureToGraph(a->stream, body, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed));
        int rc = amr_enqueue_correction(a, &count);
        amr_enqueue_residual(a, &count, true);
        solve_decide_kernel<<<1, 32, 0, a->stream>>>(handle, a->d_loop, a->d_norm + 2);
        ++count;
        cudaError_t e = cudaStreamEndCapture(a->stream, &dummy);
        if (rc != VMG_OK) return rc;
        AMR_TRY(a, e);
        AMR_TRY(a, cudaGraphInstantiate(&a->loop_exec, g, 0));
        a->loop_launches = count;
    }
    const int max = (int)a->h_loop[2];
    AMR_TRY(a, cudaMemcpyAsync(a->d_loop, a->h_loop, 9 * sizeof(double), cudaMemcpyHostToDevice, a->stream));
    AMR_TRY(a, cudaGraphLaunch(a->loop_exec, a->stream));
    AMR_TRY(a, cudaMemcpyAsync(a->h_loop, a->d_loop, (size_t)(8 + max + 1) * sizeof(double), cudaMemcpyDeviceToHost, a->stream));
    AMR_TRY(a, cudaStreamSynchronize(a->stream));
    return VMG_OK;
}

}  // namespace

extern "C" {

int vmg_amr_destroy(vmg_amr_handle a)
{
    if (!a) return VMG_ERR_ARG;
    if (a->stream) cudaStreamSynchronize(a->stream);
    amr_drop_graphs(a);
    for (vmg_s* h : a->hf) if (h) vmg_destroy(h);   // the patches first: the coarse handle may own the stream
    if (a->hc) vmg_destroy(a->hc);
    for (cudaStream_t s : a->ps) cudaStreamDestroy(s);
    for (cudaEvent_t e : a->ev_join) cudaEventDestroy(e);
    if (a->ev_fork) cudaEventDestroy(a->ev_fork);
    if (a->base) cudaFree(a->base);
    if (a->h_norm) cudaFreeHost(a->h_norm);
    if (a->h_loop) cudaFreeHost(a->h_loop);
    (void)cudaGetLastError();
    delete a;
    return VMG_OK;
}

int vmg_amr_create(vmg_amr_handle* out, int nx, int ny, int nz, double dx, double dy, double dz,
                   int npatch, const int* lo, const int* hi, void* cuda_stream)
{
    if (!out || !lo || !hi || npatch < 1) return VMG_ERR_ARG;
    *out = nullptr;
    const int n[3] = {nx, ny, nz}, nd = nz > 1 ? 3 : 2;
    for (int q = 0; q < npatch; ++q)
        for (int d = 0; d < nd; ++d)   // A1: inside the box, one coarse cell away from its boundary, at least two coarse cells wide
            if (lo[3 * q + d] < 1 || hi[3 * q + d] > n[d] - 1 || hi[3 * q + d] - lo[3 * q + d] < 2) return VMG_ERR_SIZE;
    for (int q = 0; q < npatch; ++q)       // A1: two patches at least two coarse cells apart in some direction
        for (int r = q + 1; r < npatch; ++r) {
            bool apart = false;
            for (int d = 0; d < nd; ++d)
                apart = apart || lo[3 * r + d] - hi[3 * q + d] >= 2 || lo[3 * q + d] - hi[3 * r + d] >= 2;
            if (!apart) return VMG_ERR_SIZE;
        }
    vmg_amr_s* a = new (std::nothrow) vmg_amr_s();
    if (!a) return VMG_ERR_ALLOC;
    int rc = vmg_create(&a->hc, nx, ny, nz, dx, dy, dz, cuda_stream);
    if (rc != VMG_OK) { vmg_amr_destroy(a); return rc; }
    a->stream = a->hc->stream;
    const VmgLevel& C0 = a->hc->lev[0];
    const size_t arr = (size_t)C0.nalloc + 2 * (size_t)C0.pad;
    size_t total = round_up(arr, 32) + 32 + round_up(8 + kLoopMaxCycles + 1, 32);
    for (int q = 0; q < npatch; ++q) {
        int m[3] = {1, 1, 1};
        for (int d = 0; d < nd; ++d) m[d] = 2 * (hi[3 * q + d] - lo[3 * q + d]);
        vmg_s* hf = nullptr;
        cudaStream_t sq = a->stream;
        if (npatch > 1) {
            cudaEvent_t ev = nullptr;
            if (cudaStreamCreateWithFlags(&sq, cudaStreamNonBlocking) != cudaSuccess ||
                cudaEventCreateWithFlags(&ev, cudaEventDisableTiming) != cudaSuccess) {
                (void)cudaGetLastError();
                vmg_amr_destroy(a);
                return VMG_ERR_CUDA;
            }
            a->ps.push_back(sq); a->ev_join.push_back(ev);
        }
        // two levels only (the patch itself and its shadow): any even patch size is legal, whatever its coarser grids would be
        rc = create_impl(&hf, m[0], m[1], m[2], 0.5 * dx, 0.5 * dy, nd == 3 ? 0.5 * dz : dz, (void*)sq, nullptr, 0, nullptr, 2);
        if (rc == VMG_OK) a->hf.push_back(hf);
        if (rc == VMG_OK && hf->nlev < 2) rc = VMG_ERR_SIZE;
        if (rc != VMG_OK) { vmg_amr_destroy(a); return rc; }
        hf->l2_persist_mb = 0.0;            // one stream: the access-policy window belongs to the coarse box
        AmrGeom A;
        A.C = C0.G; A.F = hf->lev[0].G; A.S = hf->lev[1].G; A.nd = nd;
        for (int d = 0; d < 3; ++d) { A.lo[d] = d < nd ? lo[3 * q + d] : 0; A.hi[d] = d < nd ? hi[3 * q + d] : 1; }
        a->A.push_back(A);
        total += round_up((size_t)hf->lev[0].n, 32) + round_up((size_t)hf->lev[1].n, 32);
    }
    a->epoch_f.assign((size_t)npatch, 0u);
    if (npatch > 1 && cudaEventCreateWithFlags(&a->ev_fork, cudaEventDisableTiming) != cudaSuccess) {
        (void)cudaGetLastError();
        vmg_amr_destroy(a);
        return VMG_ERR_CUDA;
    }
    if (cudaMalloc(&a->base, total * sizeof(double)) != cudaSuccess ||
        cudaMallocHost((void**)&a->h_norm, 4 * sizeof(double)) != cudaSuccess ||
        cudaMallocHost((void**)&a->h_loop, (8 + kLoopMaxCycles + 1) * sizeof(double)) != cudaSuccess ||
        cudaMemsetAsync(a->base, 0, total * sizeof(double), a->stream) != cudaSuccess ||
        cudaStreamSynchronize(a->stream) != cudaSuccess) {
        (void)cudaGetLastError();
        vmg_amr_destroy(a);
        return VMG_ERR_ALLOC;
    }
    double* b = (double*)a->base;
    a->btc = b + C0.pad;
    double* p = b + round_up(arr, 32);
    for (int q = 0; q < npatch; ++q) {
        a->rhsf.push_back(p); p += round_up((size_t)a->hf[q]->lev[0].n, 32);
        a->old.push_back(p);  p += round_up((size_t)a->hf[q]->lev[1].n, 32);
    }
    a->d_norm = (unsigned long long*)p;
    a->d_loop = p + 8;
    *out = a;
    return VMG_OK;
}

int vmg_amr_num_patches(vmg_amr_handle a) { return a ? a->np() : VMG_ERR_ARG; }

int vmg_amr_fine_dims(vmg_amr_handle a, int patch, int dims[3])
{
    if (!a || !dims || patch < 0 || patch >= a->np()) return VMG_ERR_ARG;
    dims[0] = a->A[patch].F.nx; dims[1] = a->A[patch].F.ny; dims[2] = a->A[patch].F.nz;
    return VMG_OK;
}

int vmg_amr_set_coeffs(vmg_amr_handle a, const double* a_c, const double* bx_c, const double* by_c, const double* bz_c,
                       const double* const* a_f, const double* const* bx_f, const double* const* by_f, const double* const* bz_f,
                       double alpha, double beta)
{
    if (!a) return VMG_ERR_ARG;
    for (int q = 0; q < a->np(); ++q)                      // the absorption term exists on both levels or on neither
        if (!a_c != !(a_f && a_f[q])) return VMG_ERR_ARG;
    int rc = vmg_set_coeffs(a->hc, a_c, bx_c, by_c, bz_c, alpha, beta);
    if (rc != VMG_OK) { a->last_cuda_error = a->hc->last_cuda_error; return rc; }
    for (int q = 0; q < a->np(); ++q) {
        vmg_s* hf = a->hf[q];
        rc = vmg_set_coeffs(hf, a_f ? a_f[q] : nullptr, bx_f ? bx_f[q] : nullptr, by_f ? by_f[q] : nullptr, bz_f ? bz_f[q] : nullptr, alpha, beta);
        if (rc != VMG_OK) { a->last_cuda_error = hf->last_cuda_error; return rc; }
        // A2: the patch's faces carry beta b / (1.5 hf^2) = 2 * (beta b / hf^2) / 3: scale its boundary planes, then 1/D again
        VmgLevel& F0 = hf->lev[0];
        for (int f = 0; f < 2 * a->A[q].nd; ++f) {
            const long long npl = (long long)plane_count(F0, f);
            amr_scale_kernel<<<grid_for(npl), kThreads, 0, hf->stream>>>(F0.wb[f], npl, 1.0 / 3.0);
        }
        hf->dinv_dirty = true;
    }
    AMR_TRY(a, cudaGetLastError());
    a->have_coeffs = true;
    return VMG_OK;
}

int vmg_amr_set_bc(vmg_amr_handle a, const int type[6], const double* const value[6])
{
    if (!a || !type) return VMG_ERR_ARG;
    int rc = vmg_set_bc(a->hc, type, value);
    if (rc != VMG_OK) return rc;
    const int all_dirichlet[6] = {VMG_BC_DIRICHLET, VMG_BC_DIRICHLET, VMG_BC_DIRICHLET, VMG_BC_DIRICHLET, VMG_BC_DIRICHLET, VMG_BC_DIRICHLET};
    for (int q = 0; q < a->np(); ++q) {
        rc = vmg_set_bc(a->hf[q], all_dirichlet, nullptr);
        if (rc != VMG_OK) return rc;
        for (int f = 0; f < 2 * a->A[q].nd; ++f) a->hf[q]->bc_has_value[f] = true;   // the planes are written by amr_ghost_kernel
    }
    a->have_bc = true;
    return VMG_OK;
}

int vmg_amr_set_option(vmg_amr_handle a, const char* key, double v)
{
    if (!a || !key) return VMG_ERR_ARG;
    if (!strcmp(key, "nu_f")) { if (v < 1 || v > 64) return VMG_ERR_ARG; a->nu_f = (int)v; return VMG_OK; }
    return vmg_set_option(a->hc, key, v);
}

int vmg_amr_get_info(vmg_amr_handle a, int* cycles, double* relres, double* history)
{
    if (!a) return VMG_ERR_ARG;
    if (cycles) *cycles = a->cycles;
    if (relres) *relres = a->relres;
    if (history) memcpy(history, a->hist.data(), a->hist.size() * sizeof(double));
    return VMG_OK;
}

// vmg_debug_pad_check over all handles (the zero pads and pad elements of every level array of the box and of the patches)
int vmg_amr_debug_pad_check(vmg_amr_handle a, long long* nonzero)
{
    if (!a || !nonzero) return VMG_ERR_ARG;
    long long total = 0, one = 0;
    int rc = vmg_debug_pad_check(a->hc, &total);
    for (int q = 0; q < a->np() && rc == VMG_OK; ++q) { rc = vmg_debug_pad_check(a->hf[q], &one); total += one; }
    *nonzero = total;
    return rc;
}

long long vmg_amr_last_launch_count(vmg_amr_handle a) { return a ? a->launches : 0; }
int vmg_amr_last_cuda_error(vmg_amr_handle a) { return a ? a->last_cuda_error : 0; }

int vmg_amr_solve(vmg_amr_handle a, const double* rhs_c, const double* const* rhs_f, double* phi_c, double* const* phi_f,
                  double rtol, int max_cycles)
{
    if (!a || !rhs_c || !rhs_f || !phi_c || !phi_f || max_cycles < 0) return VMG_ERR_ARG;
    for (int q = 0; q < a->np(); ++q) if (!rhs_f[q] || !phi_f[q]) return VMG_ERR_ARG;
    if (!a->have_coeffs || !a->have_bc) return VMG_ERR_STATE;
    vmg_s* hc = a->hc;
    int rc = ready(hc);
    for (int q = 0; q < a->np() && rc == VMG_OK; ++q) rc = ready(a->hf[q]);
    if (rc != VMG_OK) return rc;
    VmgLevel& C0 = hc->lev[0];
    a->hist.clear(); a->cycles = 0; a->relres = 0.0; a->launches = 0;
    // begin: btilde_c (box boundary values folded, zero under the patches), the two norms of A5, phi into the internal layouts
    AMR_TRY(a, cudaMemsetAsync(a->d_norm, 0, 4 * sizeof(unsigned long long), a->stream));
    rc = enqueue_fold_bc(hc, rhs_c, a->btc);
    if (rc != VMG_OK) return rc;
    long long count = 2;
    for (int q = 0; q < a->np(); ++q)
        amr_mask_norm_kernel<<<grid_for(C0.n), kThreads, 0, a->stream>>>(a->A[q], a->btc, q == a->np() - 1 ? a->d_norm + 0 : nullptr);
    count += a->np();
    // rhs' of the coarse V-cycle = btilde_c except in and next to the patches (rewritten every cycle)
    AMR_TRY(a, cudaMemcpyAsync(C0.rhs, a->btc, (size_t)C0.nalloc * sizeof(double), cudaMemcpyDeviceToDevice, a->stream));
    to_internal_kernel<<<conv_grid(C0.n), kThreads, 0, a->stream>>>(C0.G, phi_c, C0.phi, nullptr);
    amr_fork(a);
    for (int q = 0; q < a->np(); ++q) {      // per patch, on its stream (ghosts read uncovered coarse cells only)
        vmg_s* hf = a->hf[q];
        VmgLevel& F0 = hf->lev[0];
        cudaStream_t sq = amr_pstream(a, q);
        norm_inf_kernel<<<std::min<unsigned>(grid_for(F0.n), 4u * hf->num_sms), kThreads, 0, sq>>>(rhs_f[q], F0.n, a->d_norm + 1);
        cudaMemcpyAsync(a->rhsf[q], rhs_f[q], (size_t)F0.n * sizeof(double), cudaMemcpyDeviceToDevice, sq);
        to_internal_kernel<<<conv_grid(F0.n), kThreads, 0, sq>>>(F0.G, phi_f[q], F0.phi, nullptr);
        amr_average_down_kernel<<<grid_for(a->A[q].S.n), kThreads, 0, sq>>>(a->A[q], F0.phi, C0.phi, a->old[q]);
        count += 3;
        int r1 = amr_enqueue_ghost_fold(a, q, &count);
        if (r1 != VMG_OK) rc = r1;
    }
    amr_join(a);
    if (rc != VMG_OK) return rc;
    a->launches += count;
    AMR_TRY(a, cudaGetLastError());
    int status = VMG_MAXCYCLES, slow = 0;
    double nb = 0.0;
    const int tail = hc->tail_level < 0 ? hc->nlev - 1 : hc->tail_level;
    const bool red_ok = hc->nu2 >= 1 && !hc->symmetric && tail > 0;   // after a V-cycle the box was last touched by a black half-sweep (R12)
    for (int c = 0;; ++c) {
        rc = amr_run(a, c > 0 && red_ok ? 2 : 0);
        if (rc != VMG_OK) return rc;
        AMR_TRY(a, cudaMemcpyAsync(a->h_norm, a->d_norm, 4 * sizeof(double), cudaMemcpyDeviceToHost, a->stream));
        AMR_TRY(a, cudaStreamSynchronize(a->stream));
        if (c == 0) {
            nb = std::max(a->h_norm[0], a->h_norm[1]);
            if (std::isnan(a->h_norm[0]) || std::isnan(a->h_norm[1])) nb = a->h_norm[0] + a->h_norm[1];
            if (nb == 0.0) {                               // zero data: phi = 0
                AMR_TRY(a, cudaMemsetAsync(phi_c, 0, (size_t)C0.n * sizeof(double), a->stream));
                for (int q = 0; q < a->np(); ++q)          // (on the main stream: nothing is in flight on the patch streams)
                    AMR_TRY(a, cudaMemsetAsync(phi_f[q], 0, (size_t)a->hf[q]->lev[0].n * sizeof(double), a->stream));
                AMR_TRY(a, cudaStreamSynchronize(a->stream));
                a->hist.push_back(0.0);
                return VMG_OK;
            }
        }
        a->relres = a->h_norm[2] / nb;
        a->hist.push_back(a->relres);
        a->cycles = c;
        if (std::isnan(a->relres) || std::isinf(a->relres)) { status = VMG_ERR_DIVERGED; break; }
        if (rtol > 0.0) {
            if (a->relres <= rtol) { status = VMG_OK; break; }
            if (c > 0) {
                slow = (a->hist[c] >= 0.9 * a->hist[c - 1]) ? slow + 1 : 0;
                if (slow >= 3) { status = VMG_STALLED; break; }
            }
        }
        if (c == max_cycles) { status = VMG_MAXCYCLES; break; }
        if (c == 0 && red_ok && hc->use_loop && hc->use_graph && !hc->profile && max_cycles <= kLoopMaxCycles) {
            // the remaining cycles in one graph launch with the exit rules on the device
            if (!amr_graphs_current(a)) { rc = amr_run(a, -1); if (rc != VMG_OK) return rc; }   // (re)capture the three plain graphs first: they carry the epochs
            double* st = a->h_loop;
            st[0] = nb; st[1] = rtol; st[2] = (double)max_cycles; st[3] = 0.0; st[4] = 0.0; st[5] = (double)VMG_MAXCYCLES;
            st[6] = st[7] = 0.0; st[8] = a->relres;
            rc = amr_run_loop(a);
            if (rc != VMG_OK) return rc;
            const int done = (int)st[3];
            for (int i = 1; i <= done; ++i) a->hist.push_back(st[8 + i]);
            a->cycles = done; a->relres = a->hist.back();
            a->launches += (long long)done * a->loop_launches;
            status = (int)st[5];
            break;
        }
        rc = amr_run(a, 1);
        if (rc != VMG_OK) return rc;
    }
    if (status >= 0) {
        to_natural_kernel<<<conv_grid(C0.n), kThreads, 0, a->stream>>>(C0.G, C0.phi, phi_c);
        amr_fork(a);
        for (int q = 0; q < a->np(); ++q) {
            VmgLevel& F0 = a->hf[q]->lev[0];
            to_natural_kernel<<<conv_grid(F0.n), kThreads, 0, amr_pstream(a, q)>>>(F0.G, F0.phi, phi_f[q]);
        }
        amr_join(a);
        a->launches += 1 + a->np();
        AMR_TRY(a, cudaGetLastError());
    }
    AMR_TRY(a, cudaStreamSynchronize(a->stream));
    return status;
}

}  // extern "C"
