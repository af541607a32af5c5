// vmg_internal.h -- data structures of libvmg (CUDA side only; shares nothing with oracle/).
//
// Internal stencil form of a level (built by vmg_set_coeffs / vmg_set_bc):
//   wx[c] = beta*bx/hx^2 of the LOW-x face of cell c, stored per cell and 0 where that face is a domain
//           boundary; the HIGH-x face weight of cell c is the wx of its high-x neighbour (a zero pad element
//           after the last cell of a row).  Same for wy (one row on) and wz (one plane on).
//   Cell arrays are stored x-parity split (struct Geom in vmg_kernels.cuh): per row the even-x cells, a zero,
//   the odd-x cells, a zero.
//   dinv[c] = 1 / D_c,  D_c = alpha*a_c + sum(interior face weights) + 2*sum(Dirichlet boundary face weights)
//   dbase[c] = alpha*a_c + sum(interior face weights)          (boundary-type independent part of D_c)
//   wb[f]    = boundary-face weights beta*b/h^2 on domain face f (a plane), used to finish dinv and by fold_bc
// Every cell array is allocated with `pad` zeroed doubles before and after, so that the six neighbours of every
// cell are always readable and every out-of-domain neighbour is multiplied by a zero weight:
// the kernels carry no boundary branches (PAPER.md:230,266,284 boundary kinds live in the coefficients).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cstdint>
#include <vector>
#include "vmg_kernels.cuh"

// kernel classes for the optional per-kernel event profile (vmg_get_profile)
enum { VMG_PC_SMOOTH0 = 0, VMG_PC_RESREST0 = 1, VMG_PC_PROLONG0 = 2, VMG_PC_COARSE = 3, VMG_PC_NORM = 4,
       VMG_PC_FOLD = 5, VMG_PC_COPY = 6, VMG_PC_SETUP = 7, VMG_PC_COUNT = 8 };

struct VmgProfEvent { int cls; long long launches; cudaEvent_t start, stop; };

// a cached TMA descriptor of one level array for one box shape (vmg_sched.cuh level_map)
struct VmgTensorMap { const double* base; int nxp, nyt, rank; alignas(64) CUtensorMap map; };

constexpr int kLoopMaxCycles = 1000;   // longest solve the device-side loop keeps a history for (longer ones: host loop)

struct VmgLevel {
    int nx = 0, ny = 0, nz = 0;
    long long n = 0;          // cells
    vmg::Geom G;              // internal layout of the cell arrays
    long long nalloc = 0;     // doubles of one cell array (pitch * ny * nz)
    long long pad = 0;        // zeroed doubles before and after each padded array
    double hx = 0, hy = 0, hz = 0;
    // padded cell arrays (pointer to cell 0)
    double *wx = nullptr, *wy = nullptr, *wz = nullptr, *dinv = nullptr, *dbase = nullptr;
    double *phi = nullptr, *rhs = nullptr;
    double *phi2 = nullptr;   // second phi buffer: passes of the blocked smoother ping-pong (tiles overlap)
    int dir = 0;              // direction of the next whole-level kernel (see next_dir)
    int cur = 0;              // which buffer holds phi while a V-cycle is being enqueued (0: phi, 1: phi2)
    bool first_red_done = false;   // while a V-cycle is being enqueued: the finer level's restriction has already stored this level's first red half-sweep
    // boundary-face weight planes, order XLO..ZHI (unpadded)
    double* wb[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    // averaged raw coefficients in the public layout (levels >= 1 only; level 0 reads the caller's arrays)
    double *a = nullptr, *bx = nullptr, *by = nullptr, *bz = nullptr;
    double cx = 0.0, cy = 0.0, cz = 0.0;   // beta / h^2 of this level
    int cw = 0;                             // constant face weights (LevelView::cw: 0 arrays, 1 constant, 2 constant + mask)
    const unsigned char* mk = nullptr;      // cw == 2: the open faces of every cell, one byte, internal layout
    double* adiag = nullptr;  // masking: extra diagonal of this level, public layout (nullptr without a mask)
    std::vector<VmgTensorMap> tmaps;   // TMA descriptors of this level's arrays (blocked smoother, vmg_block3.cuh)
    // set only while the batched coarse segment of a vmg_create_batch group is being captured (vmg_sched.cuh): the launches of
    // this level then run over nprob problems whose arrays lie pstride doubles apart
    int nprob = 1;
    long long pstride = 0;
};

struct vmg_s;

// K handles created together (vmg_create_batch): one arena allocation, member k's arena k * stride bytes after member 0's,
// one stream.  The coarser levels of all members run as single launches (kernel-level batching).
struct VmgBatchGroup {
    void* base = nullptr;
    size_t stride_bytes = 0;
    int refs = 0;
    std::vector<vmg_s*> members;
    cudaGraph_t coarse_graph = nullptr;          // levels 1.. of ALL members: strokes + tail, problem-major launches
    cudaGraphExec_t coarse_exec = nullptr;
    std::vector<unsigned> coarse_epochs;         // the members' graph epochs the graph was captured at
    long long coarse_launches = 0;
    cudaGraph_t full_graph = nullptr;            // all levels of ALL members + their residual norms (small grids: K working sets share the L2)
    cudaGraphExec_t full_exec = nullptr;
    std::vector<unsigned> full_epochs;
    long long full_launches = 0;
    cudaStream_t owned_stream = nullptr;         // a stream the library created for the group (destroyed with the last member)
};

struct vmg_s {
    VmgBatchGroup* group = nullptr;
    int group_index = 0;
    int nlev = 0;
    bool three_d = true;
    std::vector<VmgLevel> lev;
    cudaStream_t stream = nullptr;
    bool own_stream = false;
    int device = 0;
    int num_sms = 0;
    double alpha = 0.0, beta = 1.0;
    int bctype[6] = {1, 1, 1, 1, 1, 1};
    double* bcval[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};   // device copies of value planes
    bool bc_has_value[6] = {false, false, false, false, false, false};
    bool have_coeffs = false, have_bc = false, dinv_dirty = true;
    int nu1 = 3, nu2 = 3, nbottom = 32;
    int const_weights = 1;                  // option "const_weights": use the constant-weight kernels when b == NULL
    double cw_beta = -1.0;                  // beta of the last vmg_set_coeffs with b == NULL (the captured constant-weight graphs carry beta/h^2 by value)
    int prolong = 0;              // 0: piecewise constant (R9 default), 1: trilinear
    int symmetric = 0;            // 1: symmetric V-cycle (post-smoothing / second half of the bottom black -> red): the PCG preconditioner
    int use_graph = 1, use_blocked = 0;   // blocked passes: measured slower than per-colour launches on B200
    double l2_persist_mb = 24.0;  // L2 set aside for the level-0 face weights (0: none); see apply_l2_window
    bool l2_applied = false, l2_window_set = false;
    cudaStreamAttrValue l2_attr = {};   // the window as set on the stream (members of a batch group share a stream and re-apply theirs before a capture)
    bool l2_limit_saved = false;  // cudaLimitPersistingL2CacheSize as it was before this handle raised it (restored by vmg_destroy)
    size_t l2_limit_prev = 0;
    int use_pdl = 1;              // programmatic dependent launch of the V-cycle kernels
    long long phi_keep_cells = 1ll << 25;     // option "phi_keep_cells": levels with at least this many cells (default 32 Mi: phi = 2 x L2) load the neighbours' phi with the normal policy
    int snake = 1;                // consecutive half-sweeps walk the level in opposite directions (L2 reuse)
    int use_tail = 1;             // run the coarsest levels in one CTA (vmg_tail.cuh)
    int tail_level = -1;          // first level handled by the single-CTA coarse tail (-1: none)
    size_t tail_smem = 0;         // dynamic shared memory of the tail kernel
    int use_cluster = 1;          // option "cluster": the level above the tail distributed over a thread-block cluster (vmg_cluster.cuh)
    int cl_nc = 0, cl_P = 0;      // cluster size (0: not used) and planes per CTA; tail_level is then the distributed level
    size_t cl_smem = 0;
    long long block_min_cells = 4096;   // smallest level the blocked smoother is used on
    int use_bottom_matrix = 1;    // option "bottom_matrix": the single-CTA tail applies the bottom solve as a matrix (vmg_tail.cuh bottom_matrix_kernel)
    double* bottom_S = nullptr;   // that matrix (arena; kBottomMatrixMax squared doubles)
    bool bottom_dirty = true;     // coefficients, boundary types or bottom_sweeps changed since it was built
    long long restrict_red_cells = 1ll << 18;   // option "restrict_red_cells": levels with at least this many cells restrict the red children's residuals only after a pre-smoothing (vmg_kernels.cuh restrict_one)
    double batch_full_mb = 400.0;  // option "batch_full_mb" (member 0 of a vmg_create_batch group): all levels batched while K fine levels (56 B/cell) stay below this
    // device scalars
    double* d_scal = nullptr;     // [0] = ||btilde||_inf bits, [1] = residual norm bits, ...
    double* h_scal = nullptr;     // pinned host mirror
    // arena
    void* arena = nullptr;
    size_t arena_bytes = 0;
    bool own_arena = true;        // false: a slice of a vmg_create_batch allocation
    // graph of one V-cycle (+ residual norm)
    // one slot per kind of level-0 kernels (LevelView::cw), so that a time step that alternates
    // between the two kinds of equation re-instantiates nothing; a slot is current when its epoch equals graph_epoch
    cudaGraph_t graph[3] = {nullptr, nullptr, nullptr};
    cudaGraphExec_t graph_exec[3] = {nullptr, nullptr, nullptr};
    unsigned graph_slot_epoch[3] = {0, 0, 0};
    long long graph_slot_launches[3] = {0, 0, 0};
    // the whole cycle loop of vmg_solve as ONE graph with a conditional WHILE node (run_solve_loop in vmg_sched.cuh): the
    // exit rules run on the device, the residual norm rides on the first half-sweep of the next cycle
    int use_loop = 1;                  // option "device_loop"
    cudaGraph_t loop_graph[3] = {nullptr, nullptr, nullptr};
    cudaGraphExec_t loop_exec[3] = {nullptr, nullptr, nullptr};
    unsigned loop_epoch[3] = {0, 0, 0};
    long long loop_launches_head[3] = {0, 0, 0}, loop_launches_body[3] = {0, 0, 0};
    double* d_loop = nullptr;          // device: nb, rtol, max, cycles, slow, status, -, -, hist[kLoopMaxCycles + 1]
    double* h_loop = nullptr;          // pinned host mirror
    // the same cycle cut in three graphs for the staggered batch schedule (vmg_solve_batch): [cw][segment], segment
    // 0 = level-0 down-stroke, 1 = all coarser levels, 2 = level-0 up-stroke + residual norm
    cudaGraph_t seg_graph[3][3] = {};
    cudaGraphExec_t seg_exec[3][3] = {};
    long long seg_launches[3][3] = {};
    unsigned seg_epoch[3] = {0, 0, 0};
    cudaEvent_t token = nullptr;       // "level 0 of the GPU is free again" (staggered batch schedule)
    cudaStream_t coarse_stream = nullptr;   // highest priority: the coarser levels of this handle beside another handle's fine level
    cudaEvent_t coarse_done = nullptr;
    // state of the solve in progress (vmg_solve / vmg_solve_batch phases)
    double sv_rtol = 0.0, sv_nb = 0.0;
    int sv_max = 0, sv_slow = 0, sv_status = 0;
    bool sv_active = false;
    double* sv_phi = nullptr;
    // cell masking (vmg_set_mask): device copies and the effective level-0 coefficients, one allocation
    void* mask_base = nullptr;
    unsigned char* d_mask = nullptr;
    unsigned char* mk0 = nullptr;      // open-face bits of level 0 in the internal layout (inside mask_base)
    double *d_cval = nullptr, *m_fold = nullptr, *m_a = nullptr, *m_bx = nullptr, *m_by = nullptr, *m_bz = nullptr;
    int mask_kind = 1;
    long long mask_covered = 0;
    // MG-preconditioned CG (vmg_solve_pcg): x, p, q in the internal layout, partial sums, device scalars; allocated on first use
    void* pcg_base = nullptr;
    double *pcg_x = nullptr, *pcg_p = nullptr, *pcg_q = nullptr, *pcg_partial = nullptr, *pcg_scal = nullptr;
    int pcg_npartial = 0;
    cudaGraph_t pcg_graph[6] = {};       // [slot + 2 * cw]
    cudaGraphExec_t pcg_exec[6] = {};
    unsigned pcg_epoch[6] = {0, 0, 0, 0, 0, 0};
    unsigned graph_epoch = 1;          // bumped whenever captured graphs become stale
    // result of the last solve
    int cycles = 0;
    double relres = 0.0;
    std::vector<double> hist;
    int last_cuda_error = 0;
    long long launches = 0;            // launches of the last solve
    long long launches_per_cycle = 0;  // kernel nodes in one V-cycle
    long long total_launches = 0;      // since vmg_create
    // optional per-kernel-class event timing (option "profile"): plain launches, one event pair per group
    bool profile = false;
    std::vector<VmgProfEvent> prof_pending;
    std::vector<cudaEvent_t> prof_pool;
    double prof_ms[VMG_PC_COUNT] = {0, 0, 0, 0, 0, 0, 0, 0};
    long long prof_launches[VMG_PC_COUNT] = {0, 0, 0, 0, 0, 0, 0, 0};
};
