// vmg_api.cu -- C-ABI boundary of libvmg (see include/vmg.h for the contract and the paper citations).
#include "../../include/vmg.h"
#include "vmg_internal.h"
#include "vmg_kernels.cuh"
#include "vmg_sched.cuh"
#include "vmg_pcg.cuh"

#include <cmath>
#include <cstring>
#include <new>

using namespace vmg;

#define CUDA_TRY(h, expr)                                                      \
    do {                                                                       \
        cudaError_t e__ = (expr);                                              \
        if (e__ != cudaSuccess) {                                              \
            if (h) (h)->last_cuda_error = (int)e__;                            \
            (void)cudaGetLastError();                                          \
            return VMG_ERR_CUDA;                                               \
        }                                                                      \
    } while (0)

static inline size_t round_up(size_t v, size_t m) { return (v + m - 1) / m * m; }

namespace {

struct ArenaPlan {
    size_t off = 0;
    size_t take(size_t doubles) { size_t o = off; off += round_up(doubles, 32); return o; }
};

size_t face_count(const VmgLevel& L, int dir)
{
    return (size_t)(L.nx + (dir == 0)) * (L.ny + (dir == 1)) * (L.nz + (dir == 2));
}

size_t plane_count(const VmgLevel& L, int f)
{
    return f < 2 ? (size_t)L.ny * L.nz : f < 4 ? (size_t)L.nx * L.nz : (size_t)L.nx * L.ny;
}

// lays the arena out; with base == nullptr only measures
size_t layout(vmg_s* h, double* base)
{
    ArenaPlan p;
    for (int l = 0; l < h->nlev; ++l) {
        VmgLevel& L = h->lev[l];
        double** padded[8] = {&L.wx, &L.wy, &L.wz, &L.dinv, &L.dbase, &L.phi, &L.rhs, &L.phi2};
        for (auto pp : padded) {
            size_t o = p.take((size_t)L.pad + (size_t)L.nalloc + (size_t)L.pad);
            if (base) *pp = base + o + L.pad;
        }
        for (int f = 0; f < 6; ++f) {
            size_t o = p.take(plane_count(L, f));
            if (base) L.wb[f] = base + o;
        }
        if (l > 0) {
            size_t o = p.take((size_t)L.n);          if (base) L.a = base + o;
            o = p.take(face_count(L, 0));            if (base) L.bx = base + o;
            o = p.take(face_count(L, 1));            if (base) L.by = base + o;
            o = p.take(face_count(L, 2));            if (base) L.bz = base + o;
        }
    }
    for (int f = 0; f < 6; ++f) {
        size_t o = p.take(plane_count(h->lev[0], f));
        if (base) h->bcval[f] = base + o;
    }
    size_t o = p.take(32);
    if (base) h->d_scal = base + o;
    o = p.take(8 + kLoopMaxCycles + 1);
    if (base) h->d_loop = base + o;
    o = p.take((size_t)kBottomMatrixMax * kBottomMatrixMax);
    if (base) h->bottom_S = base + o;
    return p.off;
}

int finalize_dinv(vmg_s* h)
{
    for (int l = 0; l < h->nlev; ++l) {
        VmgLevel& L = h->lev[l];
        DinvArgs g;
        g.dbase = L.dbase; g.dinv = L.dinv;
        for (int f = 0; f < 6; ++f) { g.wb[f] = L.wb[f]; g.dirichlet[f] = h->bctype[f] == VMG_BC_DIRICHLET; }
        g.G = L.G; g.three_d = h->three_d;
        finalize_dinv_kernel<<<grid_for(L.n), kThreads, 0, h->stream>>>(g);
    }
    CUDA_TRY(h, cudaGetLastError());
    h->dinv_dirty = false;   // (the captured V-cycle graph holds pointers and sizes only: new coefficients do not invalidate it)
    return VMG_OK;
}

bool singular(const vmg_s* h)
{
    int nd = h->three_d ? 6 : 4;
    for (int f = 0; f < nd; ++f) if (h->bctype[f] == VMG_BC_DIRICHLET) return false;
    if (h->d_mask && h->mask_kind == VMG_BC_DIRICHLET && h->mask_covered > 0) return false;   // an interior electrode pins phi
    return h->alpha == 0.0;
}

// Set part of L2 aside for the level-0 face weights (wx, wy, wz: contiguous in the arena), which every half-sweep
// re-reads: an access-policy window on the handle's stream (inherited by the captured graph nodes), hit ratio =
// set-aside / window so that the lines kept do not thrash among themselves.  Measured on 256x128x128 (B200, 126 MB
// L2): 24 MB is the optimum (-13 % on the level-0 smoother); larger carve-outs take more from the reuse
// between consecutive half-sweeps than they give.  Only when the weights do not fit L2 anyway.
int apply_l2_window(vmg_s* h)
{
    h->l2_applied = true;
    VmgLevel& L = h->lev[0];
    cudaDeviceProp prop;
    CUDA_TRY(h, cudaGetDeviceProperties(&prop, h->device));
    size_t bytes = 3 * ((size_t)L.nalloc + 2 * (size_t)L.pad) * sizeof(double);
    size_t want = (size_t)(h->l2_persist_mb * 1048576.0), cap = (size_t)prop.persistingL2CacheMaxSize;
    if (bytes < (size_t)prop.l2CacheSize / 2) want = 0;
    if (want > cap) want = cap;
    if (want == 0 && !h->l2_window_set) return VMG_OK;
    if (want) {
        if (!h->l2_limit_saved) {   // put back by vmg_destroy
            size_t prev = 0;
            if (cudaDeviceGetLimit(&prev, cudaLimitPersistingL2CacheSize) == cudaSuccess) { h->l2_limit_prev = prev; h->l2_limit_saved = true; }
            (void)cudaGetLastError();
        }
        CUDA_TRY(h, cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, want));
    }
    cudaStreamAttrValue a;
    memset(&a, 0, sizeof(a));
    if (bytes > (size_t)prop.accessPolicyMaxWindowSize) bytes = (size_t)prop.accessPolicyMaxWindowSize;
    a.accessPolicyWindow.base_ptr = (void*)(L.wx - L.pad);
    a.accessPolicyWindow.num_bytes = want ? bytes : 0;
    a.accessPolicyWindow.hitRatio = want ? (float)std::min(1.0, (double)want / (double)bytes) : 0.f;
    a.accessPolicyWindow.hitProp = cudaAccessPropertyPersisting;
    a.accessPolicyWindow.missProp = cudaAccessPropertyStreaming;
    CUDA_TRY(h, cudaStreamSetAttribute(h->stream, cudaStreamAttributeAccessPolicyWindow, &a));
    h->l2_attr = a;
    if (!want) CUDA_TRY(h, cudaCtxResetPersistingL2Cache());
    h->l2_window_set = want != 0;
    { ++h->graph_epoch; }
    return VMG_OK;
}

// the bottom grid is small enough for its solve to be kept as a matrix, and there is a bottom to speak of
bool bottom_matrix_ok(const vmg_s* h)
{
    return h->use_bottom_matrix && h->nlev >= 2 && h->lev[h->nlev - 1].n <= kBottomMatrixMax;
}

int ready(vmg_s* h)
{
    if (!h) return VMG_ERR_ARG;
    if (!h->have_coeffs || !h->have_bc) return VMG_ERR_STATE;
    prepare_blocked(h);   // once per device, outside any stream capture (every solve / step entry point passes here)
    if (!h->l2_applied) { int rc = apply_l2_window(h); if (rc != VMG_OK) return rc; }
    if (h->dinv_dirty) { int rc = finalize_dinv(h); if (rc != VMG_OK) return rc; }
    if (h->bottom_dirty && bottom_matrix_ok(h)) {   // the bottom solve as a matrix (vmg_tail.cuh), after 1/D is final
        const VmgLevel& B = h->lev[h->nlev - 1];
        bottom_matrix_kernel<<<(unsigned)B.n, kBottomMatrixMax, 0, h->stream>>>(B.wx, B.wy, B.wz, B.dinv, B.G, h->three_d ? 1 : 0, h->nbottom, h->bottom_S);
        CUDA_TRY(h, cudaGetLastError());
        h->bottom_dirty = false;
        ++h->total_launches;
    }
    return VMG_OK;
}

}  // namespace

extern "C" {

const char* vmg_strerror(int code)
{
    switch (code) {
    case VMG_OK: return "ok";
    case VMG_MAXCYCLES: return "max_vcycles reached before rtol";
    case VMG_STALLED: return "residual stalled (fp64 floor)";
    case VMG_ERR_ARG: return "invalid argument";
    case VMG_ERR_SIZE: return "grid size not supported (bottom grid > 512 cells or a dimension < 2)";
    case VMG_ERR_STATE: return "vmg_solve needs vmg_set_coeffs and vmg_set_bc first";
    case VMG_ERR_SINGULAR: return "singular problem: all faces Neumann and no absorption term";
    case VMG_ERR_DIVERGED: return "residual is NaN or Inf";
    case VMG_ERR_CUDA: return "CUDA runtime error";
    case VMG_ERR_ALLOC: return "allocation failed";
    default: return "unknown status";
    }
}

}  // extern "C"

namespace {

// slice: nullptr = allocate an arena of this handle's own; otherwise the handle lives in [slice, slice + slice_bytes)
// (vmg_create_batch) and *need receives the bytes one handle needs when slice_bytes is too small (then nothing is created)
// max_levels > 0 (the patches of the composite solve, vmg_amr.inl): at most that many levels, and no limit on the size of the
// last one -- such a handle is only smoothed, restricted and prolonged on its first two levels, never solved
int create_impl(vmg_handle* out, int nx, int ny, int nz, double dx, double dy, double dz, void* cuda_stream,
                void* slice, size_t slice_bytes, size_t* need, int max_levels = 0)
{
    if (!out) return VMG_ERR_ARG;
    *out = nullptr;
    bool three_d = nz > 1;
    if (nx < 2 || ny < 2 || nz < 1 || !(dx > 0) || !(dy > 0) || (three_d && !(dz > 0))) return VMG_ERR_SIZE;
    if ((long long)nx * ny * nz >= (1LL << 31)) return VMG_ERR_SIZE;   // kernels decompose cell numbers in 32 bits
    if (nz > 32767 || ny > 65535) return VMG_ERR_SIZE;                 // rows and planes are grid dimensions y and z (pair_launch_dims)
    int n[3] = {nx, ny, nz}, nlev = 1;
    for (;;) {   // R11: halve while every active dimension is even and stays >= 2
        bool ok = n[0] % 2 == 0 && n[0] / 2 >= 2 && n[1] % 2 == 0 && n[1] / 2 >= 2;
        if (three_d) ok = ok && n[2] % 2 == 0 && n[2] / 2 >= 2;
        if (!ok || (max_levels > 0 && nlev >= max_levels)) break;
        n[0] /= 2; n[1] /= 2; if (three_d) n[2] /= 2;
        ++nlev;
    }
    if (max_levels == 0 && (long long)n[0] * n[1] * n[2] > 512) return VMG_ERR_SIZE;
    vmg_s* h = new (std::nothrow) vmg_s();
    if (!h) return VMG_ERR_ALLOC;
    h->nlev = nlev; h->three_d = three_d;
    h->lev.resize(nlev);
    for (int l = 0; l < nlev; ++l) {
        VmgLevel& L = h->lev[l];
        L.nx = nx >> l; L.ny = ny >> l; L.nz = three_d ? nz >> l : 1;
        L.n = (long long)L.nx * L.ny * L.nz;
        L.G = make_geom(L.nx, L.ny, L.nz);
        L.nalloc = geom_alloc(L.G);
        L.pad = (long long)round_up((size_t)L.G.plane + L.G.pitch + 2, 32);
        L.hx = dx * (1 << l); L.hy = dy * (1 << l); L.hz = three_d ? dz * (1 << l) : 1.0;
    }
    cudaError_t e = cudaGetDevice(&h->device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&h->num_sms, cudaDevAttrMultiProcessorCount, h->device);
    if (e != cudaSuccess) { (void)cudaGetLastError(); delete h; return VMG_ERR_CUDA; }
    if (cuda_stream) { h->stream = (cudaStream_t)cuda_stream; h->own_stream = false; }
    else {
        // a blocking stream: ordered with the legacy default stream, and capturable into a graph
        if (cudaStreamCreate(&h->stream) != cudaSuccess) { (void)cudaGetLastError(); delete h; return VMG_ERR_CUDA; }
        h->own_stream = true;
    }
    h->arena_bytes = layout(h, nullptr) * sizeof(double);
    if (need) *need = h->arena_bytes;
    if (slice && slice_bytes >= h->arena_bytes) { h->arena = slice; h->own_arena = false; }
    else if (slice || need) {   // measuring pass of vmg_create_batch
        if (h->own_stream) cudaStreamDestroy(h->stream);
        delete h;
        return slice ? VMG_ERR_ALLOC : VMG_OK;
    }
    else if (cudaMalloc(&h->arena, h->arena_bytes) != cudaSuccess) {
        (void)cudaGetLastError();
        if (h->own_stream) cudaStreamDestroy(h->stream);
        delete h;
        return VMG_ERR_ALLOC;
    }
    layout(h, (double*)h->arena);
    if (cudaMemsetAsync(h->arena, 0, h->arena_bytes, h->stream) != cudaSuccess ||
        cudaMallocHost((void**)&h->h_scal, 32 * sizeof(double)) != cudaSuccess ||
        cudaMallocHost((void**)&h->h_loop, (8 + kLoopMaxCycles + 1) * sizeof(double)) != cudaSuccess ||
        cudaStreamSynchronize(h->stream) != cudaSuccess) {
        (void)cudaGetLastError();
        if (h->own_arena) cudaFree(h->arena);
        if (h->own_stream) cudaStreamDestroy(h->stream);
        delete h;
        return VMG_ERR_CUDA;
    }
    plan_schedule(h);
    *out = h;
    return VMG_OK;
}

}  // namespace

extern "C" {

int vmg_create(vmg_handle* out, int nx, int ny, int nz, double dx, double dy, double dz, void* cuda_stream)
{
    return create_impl(out, nx, ny, nz, dx, dy, dz, cuda_stream, nullptr, 0, nullptr);
}

// K handles for K problems on the same grid (the paper's multi-component solves), in ONE allocation with a
// constant stride between the members' arenas and on one stream: vmg_solve_batch on exactly these handles then runs the
// coarser levels of all of them as single launches (kernel-level batching); each handle is otherwise an ordinary handle.
int vmg_create_batch(int k, vmg_handle* out, int nx, int ny, int nz, double dx, double dy, double dz, void* cuda_stream)
{
    if (k < 1 || !out) return VMG_ERR_ARG;
    for (int i = 0; i < k; ++i) out[i] = nullptr;
    size_t need = 0;
    vmg_handle probe = nullptr;
    int rc = create_impl(&probe, nx, ny, nz, dx, dy, dz, cuda_stream, nullptr, 0, &need);   // sizes only
    if (rc != VMG_OK) return rc;
    VmgBatchGroup* G = new (std::nothrow) VmgBatchGroup();
    if (!G) return VMG_ERR_ALLOC;
    G->stride_bytes = round_up(need, 256);
    if (cudaMalloc(&G->base, G->stride_bytes * (size_t)k) != cudaSuccess) { (void)cudaGetLastError(); delete G; return VMG_ERR_ALLOC; }
    cudaStream_t shared = (cudaStream_t)cuda_stream;
    bool own = false;
    if (!shared) {
        if (cudaStreamCreate(&shared) != cudaSuccess) { (void)cudaGetLastError(); cudaFree(G->base); delete G; return VMG_ERR_CUDA; }
        own = true;
    }
    for (int i = 0; i < k && rc == VMG_OK; ++i) {
        rc = create_impl(&out[i], nx, ny, nz, dx, dy, dz, (void*)shared, (char*)G->base + (size_t)i * G->stride_bytes, G->stride_bytes, nullptr);
        if (rc == VMG_OK) {
            out[i]->group = G; out[i]->group_index = i;
            out[i]->own_stream = own && i == 0;      // member 0 owns a stream the library created; it is destroyed with the group
            G->members.push_back(out[i]);
            ++G->refs;
        }
    }
    if (rc != VMG_OK) {
        for (int i = 0; i < k; ++i) if (out[i]) { out[i]->own_stream = false; out[i]->group = nullptr; vmg_destroy(out[i]); out[i] = nullptr; }
        if (own) cudaStreamDestroy(shared);
        cudaFree(G->base);
        delete G;
        return rc;
    }
    G->coarse_epochs.assign((size_t)k, 0u);
    G->full_epochs.assign((size_t)k, 0u);
    return VMG_OK;
}

int vmg_destroy(vmg_handle h)
{
    if (!h) return VMG_ERR_ARG;
    cudaStreamSynchronize(h->stream);
    if (h->l2_window_set) {   // the window covers this handle's arena: take it off the (possibly caller-owned) stream
        cudaStreamAttrValue a;
        memset(&a, 0, sizeof(a));
        cudaStreamSetAttribute(h->stream, cudaStreamAttributeAccessPolicyWindow, &a);
        cudaCtxResetPersistingL2Cache();
    }
    if (h->l2_limit_saved) cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, h->l2_limit_prev);
    prof_collect(h);
    for (cudaEvent_t e : h->prof_pool) cudaEventDestroy(e);
    for (int i = 0; i < 6; ++i) {
        if (h->pcg_exec[i]) cudaGraphExecDestroy(h->pcg_exec[i]);
        if (h->pcg_graph[i]) cudaGraphDestroy(h->pcg_graph[i]);
    }
    if (h->pcg_base) cudaFree(h->pcg_base);
    if (h->mask_base) cudaFree(h->mask_base);
    for (int i = 0; i < 3; ++i) {
        if (h->loop_exec[i]) cudaGraphExecDestroy(h->loop_exec[i]);
        if (h->loop_graph[i]) cudaGraphDestroy(h->loop_graph[i]);
        if (h->graph_exec[i]) cudaGraphExecDestroy(h->graph_exec[i]);
        if (h->graph[i]) cudaGraphDestroy(h->graph[i]);
        for (int sg = 0; sg < 3; ++sg) {
            if (h->seg_exec[i][sg]) cudaGraphExecDestroy(h->seg_exec[i][sg]);
            if (h->seg_graph[i][sg]) cudaGraphDestroy(h->seg_graph[i][sg]);
        }
    }
    if (h->token) cudaEventDestroy(h->token);
    if (h->coarse_done) cudaEventDestroy(h->coarse_done);
    if (h->coarse_stream) cudaStreamDestroy(h->coarse_stream);
    if (h->h_scal) cudaFreeHost(h->h_scal);
    if (h->h_loop) cudaFreeHost(h->h_loop);
    if (h->arena && h->own_arena) cudaFree(h->arena);
    VmgBatchGroup* G = h->group;
    if (G) {   // the group's allocation, graph and (if the library created it) stream go with the last member
        for (auto& m : G->members) if (m == h) m = nullptr;
        if (G->coarse_exec) { cudaGraphExecDestroy(G->coarse_exec); G->coarse_exec = nullptr; }
        if (G->coarse_graph) { cudaGraphDestroy(G->coarse_graph); G->coarse_graph = nullptr; }
        if (G->full_exec) { cudaGraphExecDestroy(G->full_exec); G->full_exec = nullptr; }
        if (G->full_graph) { cudaGraphDestroy(G->full_graph); G->full_graph = nullptr; }
        if (h->own_stream) G->owned_stream = h->stream;
        if (--G->refs == 0) {
            cudaFree(G->base);
            if (G->owned_stream) cudaStreamDestroy(G->owned_stream);
            delete G;
        }
    }
    else if (h->own_stream) cudaStreamDestroy(h->stream);
    (void)cudaGetLastError();
    delete h;
    return VMG_OK;
}

int vmg_last_cuda_error(vmg_handle h) { return h ? h->last_cuda_error : 0; }

int vmg_set_coeffs(vmg_handle h, const double* a, const double* bx, const double* by, const double* bz,
                   double alpha, double beta)
{
    if (!h) return VMG_ERR_ARG;
    if (!bx != !by) return VMG_ERR_ARG;
    if (h->three_d && (!bx != !bz)) return VMG_ERR_ARG;
    if (!(beta > 0.0) || alpha < 0.0) return VMG_ERR_ARG;
    h->alpha = a ? alpha : 0.0;
    h->beta = beta;
    int sz = h->three_d ? 2 : 1;
    const double *fa = a, *fbx = bx, *fby = by, *fbz = h->three_d ? bz : nullptr;
    long long setup_launches = 0;
    ProfScope* ps = new ProfScope(h, VMG_PC_SETUP, &setup_launches);
    if (h->d_mask) {   // masking: level 0 is built from the effective coefficients (vmg_kernels.cuh "Cell masking")
        VmgLevel& L = h->lev[0];
        MaskArgs m;
        m.mask = h->d_mask; m.cval = h->d_cval; m.a = a; m.bx = bx; m.by = by; m.bz = h->three_d ? bz : nullptr;
        m.ea = h->m_a; m.ebx = h->m_bx; m.eby = h->m_by; m.ebz = h->m_bz; m.adiag = L.adiag; m.mfold = h->m_fold;
        m.nx = L.nx; m.ny = L.ny; m.nz = L.nz; m.three_d = h->three_d; m.dirichlet = h->mask_kind == VMG_BC_DIRICHLET;
        m.cx = beta / (L.hx * L.hx); m.cy = beta / (L.hy * L.hy); m.cz = h->three_d ? beta / (L.hz * L.hz) : 0.0;
        mask_cells_kernel<<<grid_for(L.n), kThreads, 0, h->stream>>>(m);
        mask_faces_kernel<<<grid_for((long long)face_count(L, 0)), kThreads, 0, h->stream>>>(m, 0);
        mask_faces_kernel<<<grid_for((long long)face_count(L, 1)), kThreads, 0, h->stream>>>(m, 1);
        if (h->three_d) mask_faces_kernel<<<grid_for((long long)face_count(L, 2)), kThreads, 0, h->stream>>>(m, 2);
        setup_launches += h->three_d ? 4 : 3;
        fa = a ? h->m_a : nullptr; fbx = h->m_bx; fby = h->m_by; fbz = h->three_d ? h->m_bz : nullptr;
    }
    const double* fad = h->d_mask ? h->lev[0].adiag : nullptr;
    const int cw = (!bx && h->const_weights) ? (h->d_mask ? 2 : 1) : 0;   // b = 1 on every face (LevelView::cw); with a mask: level 0 only
    if (cw) {   // the constant-weight kernels take beta/h^2 by value: graphs captured with another beta are stale.  Compared
                // with the beta of the last constant-weight call (a general call in between overwrites the levels' cx, cy, cz)
        if (h->cw_beta != beta) ++h->graph_epoch;
        h->cw_beta = beta;
    }
    for (int l = 0; l < h->nlev; ++l) {
        VmgLevel& L = h->lev[l];
        if (l > 0) {   // S0: average the previous level's raw coefficients
            launch_pdl(h, coarsen_a_kernel, grid_for(L.n), kThreads, 0, fa, L.a, L.nx, L.ny, L.nz, sz);
            launch_pdl(h, coarsen_b_kernel, grid_for((long long)face_count(L, 0)), kThreads, 0, fbx, L.bx, L.nx, L.ny, L.nz, sz, 0);
            launch_pdl(h, coarsen_b_kernel, grid_for((long long)face_count(L, 1)), kThreads, 0, fby, L.by, L.nx, L.ny, L.nz, sz, 1);
            if (h->three_d)
                launch_pdl(h, coarsen_b_kernel, grid_for((long long)face_count(L, 2)), kThreads, 0, fbz, L.bz, L.nx, L.ny, L.nz, sz, 2);
            if (fad) {   // the extra diagonal is averaged like a
                launch_pdl(h, coarsen_a_kernel, grid_for(L.n), kThreads, 0, fad, L.adiag, L.nx, L.ny, L.nz, sz);
                fad = L.adiag;
                ++setup_launches;
            }
            fa = L.a; fbx = L.bx; fby = L.by; fbz = h->three_d ? L.bz : nullptr;
            setup_launches += h->three_d ? 4 : 3;
        }
        StencilBuildArgs g;
        g.a = (l == 0 && !a) ? nullptr : fa;
        g.adiag = fad;
        g.bx = fbx; g.by = fby; g.bz = fbz;
        g.wx = L.wx; g.wy = L.wy; g.wz = L.wz; g.dbase = L.dbase;
        g.dinv = L.dinv; g.write_dinv = h->have_bc ? 1 : 0;   // boundary types known: 1/D in the same pass
        for (int f = 0; f < 6; ++f) g.dirichlet[f] = h->bctype[f] == VMG_BC_DIRICHLET;
        for (int f = 0; f < 6; ++f) g.wb[f] = L.wb[f];
        g.G = L.G; g.three_d = h->three_d;
        g.alpha = h->alpha; g.cx = beta / (L.hx * L.hx); g.cy = beta / (L.hy * L.hy);
        g.cz = h->three_d ? beta / (L.hz * L.hz) : 0.0;
        L.cx = g.cx; L.cy = g.cy; L.cz = g.cz; L.cw = cw == 2 ? (l == 0 ? 2 : 0) : cw; L.mk = l == 0 ? h->mk0 : nullptr;
        launch_pdl(h, build_stencil_kernel, grid_for(L.n), kThreads, 0, g);
        ++setup_launches;
    }
    delete ps;
    CUDA_TRY(h, cudaGetLastError());
    if (h->own_stream || h->profile) CUDA_TRY(h, cudaStreamSynchronize(h->stream));   // caller's stream: enqueue only (vmg.h, vmg_create)
    h->total_launches += setup_launches;
    if (h->profile) prof_collect(h);
    h->have_coeffs = true;
    h->dinv_dirty = !h->have_bc;
    h->bottom_dirty = true;
    return VMG_OK;
}

int vmg_set_bc(vmg_handle h, const int type[6], const double* const value[6])
{
    if (!h || !type) return VMG_ERR_ARG;
    for (int f = 0; f < 6; ++f)
        if (type[f] != VMG_BC_DIRICHLET && type[f] != VMG_BC_NEUMANN) return VMG_ERR_ARG;
    if (!h->have_bc) h->dinv_dirty = true;
    for (int f = 0; f < 6; ++f) {
        if (h->bctype[f] != type[f]) { ++h->graph_epoch; h->dinv_dirty = true; h->bottom_dirty = true; }   // the trilinear prolongation kernels carry the types by value; 1/D depends on them
        h->bctype[f] = type[f];
        bool active = f < 4 || h->three_d;
        h->bc_has_value[f] = active && value && value[f];
        if (h->bc_has_value[f])
            CUDA_TRY(h, cudaMemcpyAsync(h->bcval[f], value[f], plane_count(h->lev[0], f) * sizeof(double),
                                        cudaMemcpyDeviceToDevice, h->stream));
    }
    if (h->own_stream) CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    h->have_bc = true;
    return VMG_OK;
}

int vmg_set_mask(vmg_handle h, const unsigned char* mask, int kind, const double* cval)
{
    if (!h || (kind != VMG_BC_DIRICHLET && kind != VMG_BC_NEUMANN)) return VMG_ERR_ARG;
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    if (h->mask_base) { cudaFree(h->mask_base); h->mask_base = nullptr; }
    h->d_mask = nullptr; h->mk0 = nullptr; h->d_cval = nullptr; h->m_fold = h->m_a = h->m_bx = h->m_by = h->m_bz = nullptr;
    for (int l = 0; l < h->nlev; ++l) h->lev[l].adiag = nullptr;
    h->mask_covered = 0;
    h->have_coeffs = false;            // the stencil has to be rebuilt: vmg_set_coeffs applies the mask
    ++h->graph_epoch;
    if (!mask) return VMG_OK;
    VmgLevel& L0 = h->lev[0];
    // one allocation: [doubles: cval, m_fold, m_a, m_bx, m_by, m_bz, adiag of every level][bytes: mask]
    ArenaPlan p;
    size_t o_cval = p.take((size_t)L0.n), o_fold = p.take((size_t)L0.n), o_a = p.take((size_t)L0.n);
    size_t o_bx = p.take(face_count(L0, 0)), o_by = p.take(face_count(L0, 1)), o_bz = p.take(face_count(L0, 2));
    std::vector<size_t> o_ad((size_t)h->nlev);
    for (int l = 0; l < h->nlev; ++l) o_ad[l] = p.take((size_t)h->lev[l].n);
    size_t o_mask = p.off;
    const size_t mk_bytes = (size_t)L0.nalloc + 2 * (size_t)L0.pad;   // internal layout, pads included
    CUDA_TRY(h, cudaMalloc(&h->mask_base, o_mask * sizeof(double) + round_up((size_t)L0.n, 16) + mk_bytes));
    double* base = (double*)h->mask_base;
    h->m_fold = base + o_fold; h->m_a = base + o_a; h->m_bx = base + o_bx; h->m_by = base + o_by; h->m_bz = base + o_bz;
    for (int l = 0; l < h->nlev; ++l) h->lev[l].adiag = base + o_ad[l];
    h->d_mask = (unsigned char*)(base + o_mask);
    h->mask_kind = kind;
    CUDA_TRY(h, cudaMemcpyAsync(h->d_mask, mask, (size_t)L0.n, cudaMemcpyDeviceToDevice, h->stream));
    unsigned char* mk_base = h->d_mask + round_up((size_t)L0.n, 16);
    CUDA_TRY(h, cudaMemsetAsync(mk_base, 0, mk_bytes, h->stream));
    h->mk0 = mk_base + L0.pad;
    mask_face_bits_kernel<<<grid_for(L0.n), kThreads, 0, h->stream>>>(L0.G, h->d_mask, h->mk0);
    if (cval) {
        h->d_cval = base + o_cval;
        CUDA_TRY(h, cudaMemcpyAsync(h->d_cval, cval, (size_t)L0.n * sizeof(double), cudaMemcpyDeviceToDevice, h->stream));
    }
    // the number of covered cells decides whether a Dirichlet mask pins the solution: counted on the device, 8 bytes come back
    unsigned long long* cnt = (unsigned long long*)h->d_scal + 8;
    CUDA_TRY(h, cudaMemsetAsync(cnt, 0, sizeof(unsigned long long), h->stream));
    mask_count_covered_kernel<<<std::min<unsigned>(grid_for(L0.n), 8u * h->num_sms), kThreads, 0, h->stream>>>(h->d_mask, L0.n, cnt);
    CUDA_TRY(h, cudaMemcpyAsync(h->h_scal + 8, cnt, sizeof(unsigned long long), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    h->mask_covered = (long long)*(unsigned long long*)(h->h_scal + 8);
    return VMG_OK;
}

int vmg_set_option(vmg_handle h, const char* key, double v)
{
    if (!h || !key) return VMG_ERR_ARG;
    int iv = (int)v;
    if (!strcmp(key, "nu1")) { if (iv < 0 || iv > 8) return VMG_ERR_ARG; h->nu1 = iv; }
    else if (!strcmp(key, "nu2")) { if (iv < 0 || iv > 8) return VMG_ERR_ARG; h->nu2 = iv; }
    else if (!strcmp(key, "bottom_sweeps")) { if (iv < 1) return VMG_ERR_ARG; h->nbottom = iv; h->bottom_dirty = true; }
    else if (!strcmp(key, "bottom_matrix")) { h->use_bottom_matrix = iv != 0; h->bottom_dirty = true; }
    else if (!strcmp(key, "prolong")) { if (v != 0.0 && v != 1.0) return VMG_ERR_ARG; h->prolong = iv; }
    else if (!strcmp(key, "symmetric")) { if (v != 0.0 && v != 1.0) return VMG_ERR_ARG; h->symmetric = iv; }
    else if (!strcmp(key, "const_weights")) { h->const_weights = iv != 0; h->have_coeffs = false; }   // takes effect in vmg_set_coeffs
    else if (!strcmp(key, "graph")) { h->use_graph = iv != 0; }
    else if (!strcmp(key, "blocked")) { if (iv < 0 || iv > 3) return VMG_ERR_ARG; h->use_blocked = iv; }   // 1: vmg_block2.cuh, 2 / 3: vmg_block3.cuh (TMA; 2 x 2 patches / rows)
    else if (!strcmp(key, "tail")) { h->use_tail = iv != 0; }
    else if (!strcmp(key, "device_loop")) { h->use_loop = iv != 0; }
    else if (!strcmp(key, "cluster")) { h->use_cluster = iv != 0; }
    else if (!strcmp(key, "snake")) { h->snake = iv != 0; }
    else if (!strcmp(key, "pdl")) { h->use_pdl = iv != 0; }
    else if (!strcmp(key, "batch_full_mb")) { if (v < 0) return VMG_ERR_ARG; h->batch_full_mb = v; }
    else if (!strcmp(key, "block_min_cells")) { if (v < 0) return VMG_ERR_ARG; h->block_min_cells = (long long)v; }
    else if (!strcmp(key, "phi_keep_cells")) { if (v < 0) return VMG_ERR_ARG; h->phi_keep_cells = (long long)v; }
    else if (!strcmp(key, "restrict_red_cells")) { if (v < 0) return VMG_ERR_ARG; h->restrict_red_cells = (long long)v; }
    else if (!strcmp(key, "l2_persist")) { if (v < 0) return VMG_ERR_ARG; h->l2_persist_mb = v; h->l2_applied = false; }
    else if (!strcmp(key, "profile")) {
        h->profile = iv != 0;
        for (int c = 0; c < VMG_PC_COUNT; ++c) { h->prof_ms[c] = 0.0; h->prof_launches[c] = 0; }
    }
    else return VMG_ERR_ARG;
    { ++h->graph_epoch; }
    plan_schedule(h);
    return VMG_OK;
}

int vmg_get_info(vmg_handle h, int* cycles, double* relres, double* history)
{
    if (!h) return VMG_ERR_ARG;
    if (cycles) *cycles = h->cycles;
    if (relres) *relres = h->relres;
    if (history) memcpy(history, h->hist.data(), h->hist.size() * sizeof(double));
    return VMG_OK;
}

long long vmg_last_launch_count(vmg_handle h) { return h ? h->launches : 0; }
long long vmg_total_launch_count(vmg_handle h) { return h ? h->total_launches : 0; }

int vmg_get_profile(vmg_handle h, double ms[8], long long launches[8])
{
    if (!h) return VMG_ERR_ARG;
    for (int c = 0; c < VMG_PC_COUNT; ++c) {
        if (ms) ms[c] = h->prof_ms[c];
        if (launches) launches[c] = h->prof_launches[c];
    }
    return VMG_OK;
}

}  // extern "C"

// C5 of DESIGN.md: relres = ||btilde - A phi||_inf / ||btilde||_inf; stall rule; status codes.  The solve is cut
// into phases that only enqueue work and phases that run after a stream synchronise, so that vmg_solve_batch can
// advance several handles (one stream each) in lock-step and their kernels overlap on the GPU.
namespace {

// enqueue: fold_bc, phi -> internal layout, ||btilde||, the initial residual norm, read-back
int solve_begin(vmg_s* h, const double* rhs, double* phi, double rtol, int max_vcycles)
{
    VmgLevel& L0 = h->lev[0];
    unsigned long long* scal = (unsigned long long*)h->d_scal;
    h->hist.clear(); h->cycles = 0; h->relres = 0.0; h->launches = 0;
    h->sv_rtol = rtol; h->sv_max = max_vcycles; h->sv_phi = phi; h->sv_slow = 0; h->sv_status = VMG_MAXCYCLES; h->sv_active = false;
    // ||btilde|| is taken by fold_bc itself and max |phi_0| by the layout conversion: for a zero initial guess (every
    // cold start) the initial residual IS btilde, bit for bit (rhs + sum(w * 0) - 0 / (1/D)), and the 56 us all-cell
    // residual norm returns at once (it reads that maximum on the device: no host round trip for warm starts either).
    CUDA_TRY(h, cudaMemsetAsync(scal, 0, 4 * sizeof(double), h->stream));
    int rc = enqueue_fold_bc(h, rhs, L0.rhs, false, scal + 0);
    if (rc != VMG_OK) return rc;
    {
        ProfScope ps(h, VMG_PC_COPY, nullptr);
        to_internal_kernel<<<conv_grid(L0.n), kThreads, 0, h->stream>>>(L0.G, phi, L0.phi, h->d_mask, scal + 2);
    }
    enqueue_residual_norm(h, scal + 1, false, scal + 2);
    h->launches += 2;   // phi copy-in, first residual norm
    CUDA_TRY(h, cudaGetLastError());
    CUDA_TRY(h, cudaMemcpyAsync(h->h_scal, scal, 3 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    return VMG_OK;
}

// after a synchronise: hist[0]; sets sv_active when V-cycles are needed.  Returns a negative code on failure.
int solve_begin_finish(vmg_s* h)
{
    VmgLevel& L0 = h->lev[0];
    h->sv_nb = h->h_scal[0];
    if (h->sv_nb == 0.0) {   // zero right-hand side and homogeneous data: phi = 0
        CUDA_TRY(h, cudaMemsetAsync(h->sv_phi, 0, L0.n * sizeof(double), h->stream));
        h->hist.push_back(0.0);
        h->sv_status = VMG_OK;
        h->sv_phi = nullptr;   // nothing to copy out
        return VMG_OK;
    }
    if (h->h_scal[2] == 0.0) h->h_scal[1] = h->h_scal[0];   // zero initial guess: the residual is btilde (the norm kernel skipped itself)
    h->relres = h->h_scal[1] / h->sv_nb;
    h->hist.push_back(h->relres);
    if (std::isnan(h->relres) || std::isinf(h->relres)) { h->sv_status = VMG_ERR_DIVERGED; h->sv_phi = nullptr; return VMG_OK; }
    if (h->sv_rtol > 0.0 && h->relres <= h->sv_rtol) h->sv_status = VMG_OK;
    else h->sv_active = h->sv_max > 0;
    return VMG_OK;
}

// enqueue one V-cycle, its residual norm and the read-back
int solve_cycle_launch(vmg_s* h)
{
    unsigned long long* scal = (unsigned long long*)h->d_scal;
    int rc = run_vcycle_with_norm(h, scal + 1);       // graph replay or plain launches
    if (rc != VMG_OK) return rc;
    CUDA_TRY(h, cudaMemcpyAsync(h->h_scal + 1, scal + 1, sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    return VMG_OK;
}

// after a synchronise: exit rules
void solve_cycle_finish(vmg_s* h)
{
    const int c = ++h->cycles;
    h->relres = h->h_scal[1] / h->sv_nb;
    h->hist.push_back(h->relres);
    if (std::isnan(h->relres) || std::isinf(h->relres)) { h->sv_status = VMG_ERR_DIVERGED; h->sv_active = false; h->sv_phi = nullptr; return; }
    if (h->sv_rtol > 0.0) {
        if (h->relres <= h->sv_rtol) { h->sv_status = VMG_OK; h->sv_active = false; return; }
        h->sv_slow = (h->hist[c] >= 0.9 * h->hist[c - 1]) ? h->sv_slow + 1 : 0;
        if (h->sv_slow >= 3) { h->sv_status = VMG_STALLED; h->sv_active = false; return; }
    }
    if (c >= h->sv_max) h->sv_active = false;
}

// enqueue: phi -> the caller's array
int solve_end(vmg_s* h)
{
    VmgLevel& L0 = h->lev[0];
    if (h->sv_phi) {
        ProfScope ps(h, VMG_PC_COPY, nullptr);
        to_natural_kernel<<<conv_grid(L0.n), kThreads, 0, h->stream>>>(L0.G, L0.phi, h->sv_phi);
        h->launches += 1;
        CUDA_TRY(h, cudaGetLastError());
    }
    return VMG_OK;
}

int solve_close(vmg_s* h, int rc)
{
    if (h->profile) { cudaStreamSynchronize(h->stream); prof_collect(h); }
    h->total_launches += h->launches;
    return rc != VMG_OK ? rc : h->sv_status;
}

}  // namespace

extern "C" {

int vmg_solve(vmg_handle h, const double* rhs, double* phi, double rtol, int max_vcycles)
{
    if (!h || !rhs || !phi || max_vcycles < 0) return VMG_ERR_ARG;
    int rc = ready(h);
    if (rc != VMG_OK) return rc;
    if (singular(h)) return VMG_ERR_SINGULAR;
    rc = solve_begin(h, rhs, phi, rtol, max_vcycles);
    if (rc == VMG_OK && cudaStreamSynchronize(h->stream) != cudaSuccess) rc = VMG_ERR_CUDA;
    if (rc == VMG_OK) rc = solve_begin_finish(h);
    if (rc == VMG_OK && h->sv_active && solve_loop_ok(h, max_vcycles)) {
        // all cycles as one graph launch: WHILE node, exit rules on the device (run_solve_loop); then the same bookkeeping
        h->h_loop[0] = h->sv_nb; h->h_loop[1] = rtol; h->h_loop[2] = (double)max_vcycles; h->h_loop[3] = 0.0; h->h_loop[4] = 0.0;
        h->h_loop[5] = (double)VMG_MAXCYCLES; h->h_loop[6] = h->h_loop[7] = 0.0; h->h_loop[8] = h->hist[0];
        rc = run_solve_loop(h, (unsigned long long*)h->d_scal + 1);
        if (rc == VMG_OK && cudaStreamSynchronize(h->stream) != cudaSuccess) rc = VMG_ERR_CUDA;
        if (rc == VMG_OK) {
            const int cyc = (int)h->h_loop[3];
            for (int c = 1; c <= cyc; ++c) h->hist.push_back(h->h_loop[8 + c]);
            h->cycles = cyc;
            h->relres = h->h_loop[8 + cyc];
            h->sv_status = (int)h->h_loop[5];
            h->sv_active = false;
            if (h->sv_status == VMG_ERR_DIVERGED) h->sv_phi = nullptr;
            h->launches += h->loop_launches_head[h->lev[0].cw] + (long long)cyc * h->loop_launches_body[h->lev[0].cw];
            h->launches_per_cycle = h->loop_launches_body[h->lev[0].cw];
        }
    }
    while (rc == VMG_OK && h->sv_active) {
        rc = solve_cycle_launch(h);
        if (rc == VMG_OK && cudaStreamSynchronize(h->stream) != cudaSuccess) rc = VMG_ERR_CUDA;
        if (rc == VMG_OK) solve_cycle_finish(h);
    }
    if (rc == VMG_OK) rc = solve_end(h);
    if (cudaStreamSynchronize(h->stream) != cudaSuccess && rc == VMG_OK) rc = VMG_ERR_CUDA;
    if (rc == VMG_ERR_CUDA) { const int e = (int)cudaGetLastError(); if (e != 0 || h->last_cuda_error == 0) h->last_cuda_error = e; }   // keep the first recorded error
    return solve_close(h, rc);
}

// ---------------------------------------------------------------------------------------------------------------
// conjugate gradients preconditioned by one symmetric V-cycle (kernels: vmg_pcg.cuh)
// ---------------------------------------------------------------------------------------------------------------
}  // extern "C"

namespace {

int pcg_alloc(vmg_s* h)
{
    if (h->pcg_base) return VMG_OK;
    VmgLevel& L = h->lev[0];
    const size_t arr = round_up((size_t)L.nalloc + 2 * (size_t)L.pad, 32);
    h->pcg_npartial = (int)std::max<long long>(grid_for((long long)L.G.ne * L.ny * L.nz), 8LL * h->num_sms);   // apply / dot grids
    const size_t doubles = 3 * arr + round_up((size_t)h->pcg_npartial, 32) + 32;
    if (cudaMalloc(&h->pcg_base, doubles * sizeof(double)) != cudaSuccess) { (void)cudaGetLastError(); h->pcg_base = nullptr; return VMG_ERR_ALLOC; }
    CUDA_TRY(h, cudaMemsetAsync(h->pcg_base, 0, doubles * sizeof(double), h->stream));
    double* b = (double*)h->pcg_base;
    h->pcg_x = b + L.pad; h->pcg_p = b + arr + L.pad; h->pcg_q = b + 2 * arr + L.pad;
    h->pcg_partial = b + 3 * arr; h->pcg_scal = h->pcg_partial + round_up((size_t)h->pcg_npartial, 32);
    return VMG_OK;
}

// run `body` (which only enqueues on h->stream) as plain launches, or capture it once and replay it
template <typename F>
int pcg_run(vmg_s* h, int slot, F body)
{
    slot += 2 * h->lev[0].cw;
    if (!h->use_graph || h->profile) { body(); return cudaGetLastError() == cudaSuccess ? VMG_OK : VMG_ERR_CUDA; }
    if (h->pcg_epoch[slot] != h->graph_epoch) {
        if (h->pcg_exec[slot]) { cudaGraphExecDestroy(h->pcg_exec[slot]); h->pcg_exec[slot] = nullptr; }
        if (h->pcg_graph[slot]) { cudaGraphDestroy(h->pcg_graph[slot]); h->pcg_graph[slot] = nullptr; }
        CUDA_TRY(h, cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeRelaxed));
        body();
        cudaError_t e = cudaStreamEndCapture(h->stream, &h->pcg_graph[slot]);
        if (e == cudaSuccess) e = cudaGraphInstantiate(&h->pcg_exec[slot], h->pcg_graph[slot], 0);
        if (e != cudaSuccess) { h->last_cuda_error = (int)e; (void)cudaGetLastError(); return VMG_ERR_CUDA; }
        h->pcg_epoch[slot] = h->graph_epoch;
    }
    CUDA_TRY(h, cudaGraphLaunch(h->pcg_exec[slot], h->stream));
    return VMG_OK;
}

int solve_pcg_impl(vmg_s* h, const double* rhs, double* phi, double rtol, int max_iter)
{
    VmgLevel& L0 = h->lev[0];
    unsigned long long* scal = (unsigned long long*)h->d_scal;
    const long long n = L0.nalloc;                                   // element-wise kernels run over the whole allocation
    const unsigned gpair = grid_for((long long)L0.G.ne * L0.ny * L0.nz), glin = 8u * (unsigned)h->num_sms;
    double* r = L0.rhs;                                              // the CG residual lives where the V-cycle reads its rhs
    double* z = L0.phi;                                              // ... and z = M^-1 r where it leaves its result
    const LevelView v = view(L0);
    long long count = 0;

    int rc = enqueue_fold_bc(h, rhs, r);
    if (rc != VMG_OK) return rc;
    to_internal_kernel<<<conv_grid(L0.n), kThreads, 0, h->stream>>>(L0.G, phi, h->pcg_x, h->d_mask);
    CUDA_TRY(h, cudaMemsetAsync(scal, 0, 4 * sizeof(double), h->stream));
    norm_inf_kernel<<<glin, kThreads, 0, h->stream>>>(r, n, scal + 0);
    pcg_residual_inplace_kernel<<<gpair, kPcgThreads, 0, h->stream>>>(v, h->pcg_x, r);
    norm_inf_kernel<<<glin, kThreads, 0, h->stream>>>(r, n, scal + 1);
    h->launches += 5;
    CUDA_TRY(h, cudaGetLastError());
    CUDA_TRY(h, cudaMemcpyAsync(h->h_scal, scal, 2 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    const double nb = h->h_scal[0];
    if (nb == 0.0) {
        CUDA_TRY(h, cudaMemsetAsync(phi, 0, L0.n * sizeof(double), h->stream));
        CUDA_TRY(h, cudaStreamSynchronize(h->stream));
        h->hist.push_back(0.0);
        return VMG_OK;
    }
    h->relres = h->h_scal[1] / nb;
    h->hist.push_back(h->relres);
    if (std::isnan(h->relres) || std::isinf(h->relres)) return VMG_ERR_DIVERGED;
    int status = VMG_MAXCYCLES;
    if (rtol > 0.0 && h->relres <= rtol) status = VMG_OK;
    else if (max_iter > 0) {
        auto precondition = [&]() {                                   // z = M^-1 r: one symmetric V-cycle from zero
            cudaMemsetAsync(z - L0.pad, 0, ((size_t)L0.nalloc + 2 * (size_t)L0.pad) * sizeof(double), h->stream);
            enqueue_vcycle(h, nullptr, &count);
        };
        // p = z = M^-1 r, rho = <r, z>
        precondition();
        pcg_dot_kernel<<<glin, kPcgThreads, 0, h->stream>>>(r, z, n, h->pcg_partial);
        pcg_reduce_kernel<<<1, 1024, 0, h->stream>>>(h->pcg_partial, (int)glin, PCG_MODE_RHO0, h->pcg_scal);
        pcg_direction_kernel<<<glin, kPcgThreads, 0, h->stream>>>(h->pcg_p, z, n, h->pcg_scal, 1);
        CUDA_TRY(h, cudaGetLastError());
        h->launches += count + 3;
        const long long per_cycle = count;
        int slow = 0;
        for (int c = 1; c <= max_iter; ++c) {
            rc = pcg_run(h, 0, [&]() {                                // q = A p, alpha, x += alpha p, r -= alpha q, ||r||
                pcg_apply_dot_kernel<<<gpair, kPcgThreads, 0, h->stream>>>(v, h->pcg_p, h->pcg_q, h->pcg_partial);
                pcg_reduce_kernel<<<1, 1024, 0, h->stream>>>(h->pcg_partial, (int)gpair, PCG_MODE_ALPHA, h->pcg_scal);
                cudaMemsetAsync(scal + 1, 0, sizeof(double), h->stream);
                pcg_update_kernel<<<glin, kPcgThreads, 0, h->stream>>>(h->pcg_x, r, h->pcg_p, h->pcg_q, n, h->pcg_scal, scal + 1);
            });
            if (rc != VMG_OK) return rc;
            h->launches += 3;
            CUDA_TRY(h, cudaMemcpyAsync(h->h_scal + 1, scal + 1, sizeof(double), cudaMemcpyDeviceToHost, h->stream));
            CUDA_TRY(h, cudaStreamSynchronize(h->stream));
            h->relres = h->h_scal[1] / nb;
            h->hist.push_back(h->relres);
            h->cycles = c;
            if (std::isnan(h->relres) || std::isinf(h->relres)) return VMG_ERR_DIVERGED;
            if (rtol > 0.0) {
                if (h->relres <= rtol) { status = VMG_OK; break; }
                slow = (h->hist[c] >= 0.9 * h->hist[c - 1]) ? slow + 1 : 0;
                if (slow >= 3) { status = VMG_STALLED; break; }
            }
            if (c == max_iter) break;
            rc = pcg_run(h, 1, [&]() {                                // z = M^-1 r, beta, p = z + beta p
                long long dummy = 0;
                cudaMemsetAsync(z - L0.pad, 0, ((size_t)L0.nalloc + 2 * (size_t)L0.pad) * sizeof(double), h->stream);
                enqueue_vcycle(h, nullptr, &dummy);
                pcg_dot_kernel<<<glin, kPcgThreads, 0, h->stream>>>(r, z, n, h->pcg_partial);
                pcg_reduce_kernel<<<1, 1024, 0, h->stream>>>(h->pcg_partial, (int)glin, PCG_MODE_BETA, h->pcg_scal);
                pcg_direction_kernel<<<glin, kPcgThreads, 0, h->stream>>>(h->pcg_p, z, n, h->pcg_scal, 0);
            });
            if (rc != VMG_OK) return rc;
            h->launches += per_cycle + 3;
        }
    }
    to_natural_kernel<<<conv_grid(L0.n), kThreads, 0, h->stream>>>(L0.G, h->pcg_x, phi);
    h->launches += 1;
    CUDA_TRY(h, cudaGetLastError());
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    return status;
}

}  // namespace

extern "C" {

int vmg_solve_pcg(vmg_handle h, const double* rhs, double* phi, double rtol, int max_iter)
{
    if (!h || !rhs || !phi || max_iter < 0) return VMG_ERR_ARG;
    int rc = ready(h);
    if (rc != VMG_OK) return rc;
    if (singular(h)) return VMG_ERR_SINGULAR;
    if (h->nu1 != h->nu2) return VMG_ERR_ARG;          // the preconditioner must be symmetric
    if ((rc = pcg_alloc(h)) != VMG_OK) return rc;
    h->hist.clear(); h->cycles = 0; h->relres = 0.0; h->launches = 0;
    const int keep = h->symmetric;
    h->symmetric = 1;   // (vmg_solve's own graph is not used here and stays as captured)
    rc = solve_pcg_impl(h, rhs, phi, rtol, max_iter);
    h->symmetric = keep;
    if (h->profile) { cudaStreamSynchronize(h->stream); prof_collect(h); }
    h->total_launches += h->launches;
    return rc;
}

// N independent problems (one handle and one stream each), advanced in lock-step: every round enqueues one V-cycle
// per unfinished handle and then synchronises them, so the latency-bound coarse levels of one solve overlap the
// bandwidth-bound fine level of another (the paper's "multi-component" optimisation).
int vmg_solve_batch(int n, const vmg_handle* hs, const double* const* rhs, double* const* phi, double rtol, int max_vcycles,
                    int* status)
{
    if (n < 0 || (n > 0 && (!hs || !rhs || !phi)) || max_vcycles < 0) return VMG_ERR_ARG;
    std::vector<int> rc(n, VMG_OK);
    for (int i = 0; i < n; ++i) {
        vmg_s* h = hs[i];
        if (!h || !rhs[i] || !phi[i]) { rc[i] = VMG_ERR_ARG; continue; }
        for (int k = 0; k < i; ++k) if (hs[k] == h) rc[i] = VMG_ERR_ARG;   // a handle can run one solve at a time
        if (rc[i] != VMG_OK) continue;
        rc[i] = ready(h);
        if (rc[i] == VMG_OK && singular(h)) rc[i] = VMG_ERR_SINGULAR;
        if (rc[i] == VMG_OK) rc[i] = solve_begin(h, rhs[i], phi[i], rtol, max_vcycles);
    }
    auto sync_all = [&]() {
        for (int i = 0; i < n; ++i)
            if (rc[i] == VMG_OK && cudaStreamSynchronize(hs[i]->stream) != cudaSuccess) {
                rc[i] = VMG_ERR_CUDA; hs[i]->last_cuda_error = (int)cudaGetLastError();
            }
    };
    sync_all();
    for (int i = 0; i < n; ++i) if (rc[i] == VMG_OK) rc[i] = solve_begin_finish(hs[i]);
    for (;;) {
        bool any = false;
        // Staggered schedule: the level-0 strokes of the handles follow one another (a token event passed from stream to
        // stream), so that one handle at a time streams its fine level through the L2 -- keeping the reuse between its
        // consecutive half-sweeps -- while the latency-bound coarser levels of the others run beside it.
        int nact = 0;
        bool seg_ok = true;
        for (int i = 0; i < n; ++i)
            if (rc[i] == VMG_OK && hs[i]->sv_active) { ++nact; seg_ok = seg_ok && vcycle_segmentable(hs[i]); }
        // Kernel-level batching: the handles are exactly the members of one vmg_create_batch group (one allocation, one
        // stream).  Level 0 one problem after the other (its half-sweeps keep their L2 reuse), the coarser levels of ALL
        // members as single launches over planes x problems with K CTAs in the tail (run_group_coarse); problems that have
        // finished are simply not given their level-0 strokes any more (their coarse levels are recomputed, unused).
        VmgBatchGroup* G = n >= 2 && hs[0] ? hs[0]->group : nullptr;
        bool fused = G && (int)G->members.size() == n && nact >= 2 && seg_ok;
        for (int i = 0; fused && i < n; ++i) fused = rc[i] == VMG_OK && hs[i]->group == G;
        fused = fused && group_coarse_ok(G) && (long long)G->members[0]->lev[1].nz * n <= 65535;
        if (fused && nact == n && group_full_ok(G)) {
            // every problem still iterates and the K fine levels together fit the L2: ALL levels problem-major, one graph
            const int rcg = run_group_full(G);
            for (int i = 0; i < n; ++i) {
                vmg_s* h = hs[i];
                unsigned long long* scal = (unsigned long long*)h->d_scal;
                rc[i] = rcg;
                h->launches += G->full_launches;
                h->launches_per_cycle = G->full_launches;
                if (rc[i] == VMG_OK && cudaMemcpyAsync(h->h_scal + 1, scal + 1, sizeof(double), cudaMemcpyDeviceToHost, h->stream) != cudaSuccess) rc[i] = VMG_ERR_CUDA;
                any = true;
            }
        } else
        if (fused) {
            for (int i = 0; i < n; ++i) {
                vmg_s* h = hs[i];
                if (!h->sv_active) continue;
                rc[i] = run_vcycle_segment(h, 0, (unsigned long long*)h->d_scal + 1);
            }
            const int rcg = run_group_coarse(G);
            for (int i = 0; i < n; ++i) {
                vmg_s* h = hs[i];
                if (rc[i] != VMG_OK || !h->sv_active) continue;
                if (rcg != VMG_OK) { rc[i] = rcg; continue; }
                unsigned long long* scal = (unsigned long long*)h->d_scal;
                rc[i] = run_vcycle_segment(h, 2, scal + 1);
                h->launches += G->coarse_launches - h->seg_launches[h->lev[0].cw][1];   // the group's coarse launches in place of its own
                if (rc[i] == VMG_OK && cudaMemcpyAsync(h->h_scal + 1, scal + 1, sizeof(double), cudaMemcpyDeviceToHost, h->stream) != cudaSuccess) rc[i] = VMG_ERR_CUDA;
                any = true;
            }
        } else
        if (nact >= 2 && seg_ok) {
            cudaEvent_t prev = nullptr;
            for (int pass = 0; pass < 2; ++pass)
                for (int i = 0; i < n; ++i) {
                    vmg_s* h = hs[i];
                    if (rc[i] != VMG_OK || !h->sv_active) continue;
                    unsigned long long* scal = (unsigned long long*)h->d_scal;
                    if (!h->token) {
                        int lo = 0, hi = 0;
                        cudaDeviceGetStreamPriorityRange(&lo, &hi);
                        if (cudaEventCreateWithFlags(&h->token, cudaEventDisableTiming) != cudaSuccess ||
                            cudaEventCreateWithFlags(&h->coarse_done, cudaEventDisableTiming) != cudaSuccess ||
                            cudaStreamCreateWithPriority(&h->coarse_stream, cudaStreamNonBlocking, hi) != cudaSuccess) {
                            h->last_cuda_error = (int)cudaGetLastError(); rc[i] = VMG_ERR_CUDA; continue;
                        }
                    }
                    if (prev) cudaStreamWaitEvent(h->stream, prev, 0);
                    rc[i] = run_vcycle_segment(h, pass == 0 ? 0 : 2, scal + 1);
                    if (rc[i] != VMG_OK) continue;
                    cudaEventRecord(h->token, h->stream);
                    prev = h->token;
                    if (pass == 0) {   // the coarser levels on the high-priority stream, between the two level-0 strokes
                        cudaStreamWaitEvent(h->coarse_stream, h->token, 0);
                        rc[i] = run_vcycle_segment(h, 1, scal + 1, h->coarse_stream);
                        cudaEventRecord(h->coarse_done, h->coarse_stream);
                        cudaStreamWaitEvent(h->stream, h->coarse_done, 0);
                    }
                    else if (cudaMemcpyAsync(h->h_scal + 1, scal + 1, sizeof(double), cudaMemcpyDeviceToHost, h->stream) != cudaSuccess) rc[i] = VMG_ERR_CUDA;
                    any = true;
                }
        } else
        for (int i = 0; i < n; ++i)
            if (rc[i] == VMG_OK && hs[i]->sv_active) { rc[i] = solve_cycle_launch(hs[i]); any = true; }
        if (!any) break;
        for (int i = 0; i < n; ++i)
            if (rc[i] == VMG_OK && hs[i]->sv_active) {
                if (cudaStreamSynchronize(hs[i]->stream) != cudaSuccess) { rc[i] = VMG_ERR_CUDA; hs[i]->last_cuda_error = (int)cudaGetLastError(); }
                else solve_cycle_finish(hs[i]);
            }
    }
    for (int i = 0; i < n; ++i) if (rc[i] == VMG_OK) rc[i] = solve_end(hs[i]);
    sync_all();
    int worst = VMG_OK;
    for (int i = 0; i < n; ++i) {
        int st = rc[i];
        if (hs && hs[i] && rc[i] != VMG_ERR_ARG && rc[i] != VMG_ERR_STATE && rc[i] != VMG_ERR_SINGULAR) st = solve_close(hs[i], rc[i]);
        if (status) status[i] = st;
        if (st < 0) worst = worst < 0 ? std::min(worst, st) : st;
        else if (worst >= 0) worst = std::max(worst, st);
    }
    return worst;
}

}  // extern "C"

#include "vmg_steps.inl"
#include "vmg_amr.inl"

#ifdef VMG_TAIL_TIMING
// debug build only (-DVMG_TAIL_TIMING): clock64 stamps of the last coarse_tail_kernel launch (vmg_tail.cuh TAIL_MARK)
extern "C" int vmg_debug_tail_clock(long long* out64)
{
    return cudaMemcpyFromSymbol(out64, vmg::vmg_tail_clock, 64 * sizeof(long long)) == cudaSuccess ? 0 : -6;
}
#endif
