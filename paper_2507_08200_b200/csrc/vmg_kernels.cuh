// vmg_kernels.cuh -- baseline (one step per launch) kernels of libvmg.  fp64 throughout.
// These are the correctness baseline every fused / blocked kernel is diffed against, and they remain the
// path for levels and options the blocked kernels do not cover.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

namespace vmg {

constexpr int kThreads = 256;

__host__ __device__ inline long long cdiv(long long a, long long b) { return (a + b - 1) / b; }

// Programmatic dependent launch: the V-cycle's kernels are launched with programmaticStreamSerialization, so a kernel's
// launch (CTA scheduling, parameter fetch, index arithmetic) overlaps the tail of its predecessor; nothing of the
// predecessor's output is touched, and nothing it still reads is overwritten, before this wait (which also flushes
// the predecessor's writes).  A no-op when the kernel was launched without the attribute.
// Right after it the kernel lets ITS dependents be scheduled (the trigger fires once every CTA of this grid has started
// or exited): their CTAs fill the SM slots that this grid's last wave leaves free and sit in their own wait.
__device__ __forceinline__ void grid_dependency_wait()
{
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}

// ------------------------------------------------------------------------------------------------
// Internal layout of a level's cell arrays ("x-parity split").  A colour half-sweep
// touches every other cell of a row, so in the natural layout half of every 32-byte sector of rhs, 1/D and of the
// phi being written is fetched for nothing.  Each row therefore stores its even-x cells first, then its odd-x
// cells, each block followed by at least one zero element:   [E_0 .. E_{ne-1} 0.. | O_0 .. O_{no-1} 0..].  Each half is
// hp = ne + 1 rounded up to a multiple of 4 doubles long (pitch = 2 hp), so both halves of every row start on a 32-byte
// sector and every stride of the level is a multiple of 16 bytes: the array is then a legal TMA tensor
// (m, row pair, row parity, x-parity, plane) for the blocked smoother (vmg_block3.cuh).
// A half-sweep then reads and writes unit-stride runs and moves 5 doubles per cell of the level (10 per relaxation) instead of 7 (14).  The pad
// elements double as the zero weight / zero neighbour beyond the low and high x faces (the x-neighbours of E_m are
// O_{m-1}, O_m, those of O_m are E_m, E_{m+1}); y- and z-neighbours are +-pitch, +-plane away, and beyond the domain
// they land in another row / plane or in the zeroed pad before and after the array, always under a zero weight.
// ------------------------------------------------------------------------------------------------
struct Geom {
    int nx, ny, nz, ne, hp, pitch;   // ne = even-x cells per row, hp = doubles per half row (>= ne + 1), pitch = 2 hp
    long long plane, n;              // plane = pitch * ny (doubles per z-plane), n = nx*ny*nz (cells)
};

__host__ __device__ inline Geom make_geom(int nx, int ny, int nz)
{
    Geom G;
    G.nx = nx; G.ny = ny; G.nz = nz; G.ne = (nx + 1) / 2; G.hp = (G.ne + 1 + 3) / 4 * 4; G.pitch = 2 * G.hp;
    G.plane = (long long)G.pitch * ny; G.n = (long long)nx * ny * nz;
    return G;
}
__host__ __device__ inline long long geom_alloc(const Geom& G) { return G.plane * G.nz; }
__host__ __device__ __forceinline__ long long cell_at(const Geom& G, int i, int j, int k)
{
    return G.plane * k + (long long)G.pitch * j + (i & 1) * G.hp + (i >> 1);
}
// natural cell number t = i + nx*(j + ny*k) -> (i, j, k).  32-bit arithmetic: vmg_create caps n below 2^31, and a
// 64-bit division is ~100 dependent instructions, which the latency-bound coarse levels cannot hide.
__device__ __forceinline__ void unflatten(const Geom& G, long long t, int& i, int& j, int& k)
{
    const unsigned u = (unsigned)t, q = u / (unsigned)G.nx;
    i = (int)(u - q * (unsigned)G.nx); k = (int)(q / (unsigned)G.ny); j = (int)(q - (unsigned)k * (unsigned)G.ny);
}
// pair number t = m + ne*(j + ny*k) -> (m, j, k)
__device__ __forceinline__ void unflatten_pair(const Geom& G, long long t, int& m, int& j, int& k)
{
    const unsigned u = (unsigned)t, q = u / (unsigned)G.ne;
    m = (int)(u - q * (unsigned)G.ne); k = (int)(q / (unsigned)G.ny); j = (int)(q - (unsigned)k * (unsigned)G.ny);
}

// ------------------------------------------------------------------------------------------------
// S0. Coefficient averaging to the next coarser level (north_star (2) "coefficient averaging";
// reading R10: a = mean of children, b = mean of the fine faces lying on the coarse face).
// Public layouts on both sides.  NULL fine a means a == 0; NULL fine b means b == 1.
// ------------------------------------------------------------------------------------------------
__global__ void coarsen_a_kernel(const double* __restrict__ fa, double* __restrict__ ca,
                                 int cnx, int cny, int cnz, int sz)
{
    grid_dependency_wait();   // vmg_set_coeffs launches its kernels with programmatic serialisation
    long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    long long n = (long long)cnx * cny * cnz;
    if (t >= n) return;
    int I = (int)(t % cnx), J = (int)((t / cnx) % cny), K = (int)(t / ((long long)cnx * cny));
    int fnx = 2 * cnx, fny = 2 * cny;
    double s = 0.0;
    if (fa)
        for (int r = 0; r < sz; ++r)
            for (int q = 0; q < 2; ++q)
                for (int p = 0; p < 2; ++p)
                    s += fa[(2 * I + p) + (long long)fnx * ((2 * J + q) + (long long)fny * (sz * K + r))];
    ca[t] = s / (4.0 * sz);
}

// dir: 0 = x faces, 1 = y faces, 2 = z faces.  (cnx, cny, cnz) are coarse CELL counts.
__global__ void coarsen_b_kernel(const double* __restrict__ fb, double* __restrict__ cb,
                                 int cnx, int cny, int cnz, int sz, int dir)
{
    grid_dependency_wait();
    int ex = cnx + (dir == 0), ey = cny + (dir == 1), ez = cnz + (dir == 2);
    long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    long long n = (long long)ex * ey * ez;
    if (t >= n) return;
    int I = (int)(t % ex), J = (int)((t / ex) % ey), K = (int)(t / ((long long)ex * ey));
    int fex = 2 * cnx + (dir == 0), fey = 2 * cny + (dir == 1);
    if (!fb) { cb[t] = 1.0; return; }
    double s = 0.0;
    if (dir == 0) {
        for (int r = 0; r < sz; ++r) for (int q = 0; q < 2; ++q)
            s += fb[(2 * I) + (long long)fex * ((2 * J + q) + (long long)fey * (sz * K + r))];
        cb[t] = s / (2.0 * sz);
    } else if (dir == 1) {
        for (int r = 0; r < sz; ++r) for (int p = 0; p < 2; ++p)
            s += fb[(2 * I + p) + (long long)fex * ((2 * J) + (long long)fey * (sz * K + r))];
        cb[t] = s / (2.0 * sz);
    } else {
        for (int q = 0; q < 2; ++q) for (int p = 0; p < 2; ++p)
            s += fb[(2 * I + p) + (long long)fex * ((2 * J + q) + (long long)fey * (2 * K))];
        cb[t] = s / 4.0;
    }
}


// ------------------------------------------------------------------------------------------------
// Internal stencil form of one level from its raw coefficients (C1 of DESIGN.md).  Raw arrays in the public
// layout, internal arrays in the x-parity split layout.
// ------------------------------------------------------------------------------------------------
struct StencilBuildArgs {
    const double *a, *bx, *by, *bz;      // raw, public layout (may be NULL)
    const double* adiag;                 // masking: extra diagonal of this level, public layout (NULL without a mask)
    double *wx, *wy, *wz, *dbase;        // internal cell arrays
    double* dinv;                        // written as well when the boundary types are known (write_dinv): the same
    int write_dinv, dirichlet[6];        // expression, in the same order, as finalize_dinv_kernel
    double* wb[6];                       // boundary planes (natural plane layout)
    Geom G;
    int three_d;
    double alpha, cx, cy, cz;            // cx = beta/hx^2 ...
};

__global__ void build_stencil_kernel(StencilBuildArgs g)
{
    grid_dependency_wait();   // vmg_set_coeffs launches its kernels with programmatic serialisation
    long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t >= g.G.n) return;
    const int nx = g.G.nx, ny = g.G.ny, nz = g.G.nz;
    int i, j, k;
    unflatten(g.G, t, i, j, k);
    long long nxy = (long long)nx * ny;
    double bxl = g.bx ? g.bx[i + (long long)(nx + 1) * (j + (long long)ny * k)] : 1.0;
    double bxh = g.bx ? g.bx[i + 1 + (long long)(nx + 1) * (j + (long long)ny * k)] : 1.0;
    double byl = g.by ? g.by[i + (long long)nx * (j + (long long)(ny + 1) * k)] : 1.0;
    double byh = g.by ? g.by[i + (long long)nx * (j + 1 + (long long)(ny + 1) * k)] : 1.0;
    double wxl = g.cx * bxl, wxh = g.cx * bxh, wyl = g.cy * byl, wyh = g.cy * byh, wzl = 0.0, wzh = 0.0;
    if (g.three_d) {
        double bzl = g.bz ? g.bz[t] : 1.0;
        double bzh = g.bz ? g.bz[t + nxy] : 1.0;
        wzl = g.cz * bzl; wzh = g.cz * bzh;
    }
    double bw[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};   // this cell's boundary-face weights
    if (i == 0)      { g.wb[0][j + (long long)ny * k] = bw[0] = wxl; wxl = 0.0; }
    if (i == nx - 1) { g.wb[1][j + (long long)ny * k] = bw[1] = wxh; wxh = 0.0; }
    if (j == 0)      { g.wb[2][i + (long long)nx * k] = bw[2] = wyl; wyl = 0.0; }
    if (j == ny - 1) { g.wb[3][i + (long long)nx * k] = bw[3] = wyh; wyh = 0.0; }
    if (g.three_d) {
        if (k == 0)      { g.wb[4][i + (long long)nx * j] = bw[4] = wzl; wzl = 0.0; }
        if (k == nz - 1) { g.wb[5][i + (long long)nx * j] = bw[5] = wzh; wzh = 0.0; }
    }
    const long long c = cell_at(g.G, i, j, k);
    g.wx[c] = wxl; g.wy[c] = wyl; g.wz[c] = wzl;
    double d = g.a ? g.alpha * g.a[t] : 0.0;
    if (g.adiag) d += g.adiag[t];
    d += wxl; d += wxh; d += wyl; d += wyh; d += wzl; d += wzh;
    g.dbase[c] = d;
    if (g.write_dinv) {
        if (i == 0 && g.dirichlet[0])      d += 2.0 * bw[0];
        if (i == nx - 1 && g.dirichlet[1]) d += 2.0 * bw[1];
        if (j == 0 && g.dirichlet[2])      d += 2.0 * bw[2];
        if (j == ny - 1 && g.dirichlet[3]) d += 2.0 * bw[3];
        if (g.three_d) {
            if (k == 0 && g.dirichlet[4])      d += 2.0 * bw[4];
            if (k == nz - 1 && g.dirichlet[5]) d += 2.0 * bw[5];
        }
        g.dinv[c] = 1.0 / d;
    }
}

struct DinvArgs {
    const double* dbase; double* dinv; const double* wb[6];
    Geom G;
    int three_d; int dirichlet[6];
};

__global__ void finalize_dinv_kernel(DinvArgs g)
{
    long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t >= g.G.n) return;
    const int nx = g.G.nx, ny = g.G.ny, nz = g.G.nz;
    int i, j, k;
    unflatten(g.G, t, i, j, k);
    const long long c = cell_at(g.G, i, j, k);
    double d = g.dbase[c];
    if (i == 0 && g.dirichlet[0])      d += 2.0 * g.wb[0][j + (long long)ny * k];
    if (i == nx - 1 && g.dirichlet[1]) d += 2.0 * g.wb[1][j + (long long)ny * k];
    if (j == 0 && g.dirichlet[2])      d += 2.0 * g.wb[2][i + (long long)nx * k];
    if (j == ny - 1 && g.dirichlet[3]) d += 2.0 * g.wb[3][i + (long long)nx * k];
    if (g.three_d) {
        if (k == 0 && g.dirichlet[4])      d += 2.0 * g.wb[4][i + (long long)nx * j];
        if (k == nz - 1 && g.dirichlet[5]) d += 2.0 * g.wb[5][i + (long long)nx * j];
    }
    g.dinv[c] = 1.0 / d;
}

// ------------------------------------------------------------------------------------------------
// S1. fold_bc: btilde = f + 2*w_b*g on Dirichlet-adjacent cells + w_b*h*q on Neumann-adjacent cells
// (w_b = beta*b/h^2 of the boundary face; R3, R5).  Level 0, once per solve.  rhs: public layout; bt: internal
// layout, or public layout when bt_natural (the single-step entry point).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void block_max_to_global(double v, unsigned long long* out);

struct FoldArgs {
    unsigned long long* norm_out;                      // ||btilde||_inf accumulated here as well (S6; NULL: not wanted)
    const double* rhs; double* bt; const double* wb[6]; const double* val[6];
    const unsigned char* mask; const double* mfold;   // masking (NULL without a mask): interface terms, covered cells -> 0
    Geom G;
    int three_d, bt_natural; int dirichlet[6]; double h[3];
};

__device__ __forceinline__ double fold_bc_one(const FoldArgs& g, long long t, double v /* = g.rhs[t] */)
{
    const int nx = g.G.nx, ny = g.G.ny, nz = g.G.nz;
    int i, j, k;
    unflatten(g.G, t, i, j, k);
    auto add = [&](int f, long long pl, double hd) {
        if (!g.val[f]) return;
        double w = g.wb[f][pl], q = g.val[f][pl];
        v += g.dirichlet[f] ? 2.0 * w * q : w * hd * q;
    };
    if (i == 0)      add(0, j + (long long)ny * k, g.h[0]);
    if (i == nx - 1) add(1, j + (long long)ny * k, g.h[0]);
    if (j == 0)      add(2, i + (long long)nx * k, g.h[1]);
    if (j == ny - 1) add(3, i + (long long)nx * k, g.h[1]);
    if (g.three_d) {
        if (k == 0)      add(4, i + (long long)nx * j, g.h[2]);
        if (k == nz - 1) add(5, i + (long long)nx * j, g.h[2]);
    }
    if (g.mask) v = g.mask[t] ? v + g.mfold[t] : 0.0;
    g.bt[g.bt_natural ? t : cell_at(g.G, i, j, k)] = v;
    return v;
}

// The layout conversions (fold_bc, to_internal, to_natural) move 8 bytes per element and are bound by the bytes in flight
// (one load per thread: 2.1-3.8 TB/s): every thread takes kConvElems elements a whole grid apart, all loads issued first.
constexpr int kConvElems = 4;

__global__ void fold_bc_kernel(FoldArgs g)
{
    const long long T = (long long)gridDim.x * blockDim.x, t0 = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    double r[kConvElems];
#pragma unroll
    for (int u = 0; u < kConvElems; ++u) { const long long t = t0 + u * T; r[u] = t < g.G.n ? g.rhs[t] : 0.0; }
    double v = 0.0;
    bool nan = false;
#pragma unroll
    for (int u = 0; u < kConvElems; ++u) {
        const long long t = t0 + u * T;
        if (t < g.G.n) {
            const double x = fabs(fold_bc_one(g, t, r[u]));
            nan |= x != x;
            v = fmax(v, x);
        }
    }
    if (g.norm_out) {                                  // the same maximum norm_inf_kernel takes over the stored array
        if (nan) v = __longlong_as_double(0x7ff8000000000000ll);
        block_max_to_global(v, g.norm_out);
    }
}

// the open faces of every cell as one byte in the internal layout (LevelView::mk): bit f (0..5 = low x, high x, low y,
// high y, low z, high z) is set when the face is interior to the domain and the cells on both sides are valid
__global__ void mask_face_bits_kernel(Geom G, const unsigned char* __restrict__ nat, unsigned char* __restrict__ in)
{
    long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t >= G.n) return;
    int i, j, k;
    unflatten(G, t, i, j, k);
    const long long nxy = (long long)G.nx * G.ny;
    unsigned fb = 0;
    if (nat[t]) {
        if (i > 0 && nat[t - 1]) fb |= 1u;
        if (i < G.nx - 1 && nat[t + 1]) fb |= 2u;
        if (j > 0 && nat[t - G.nx]) fb |= 4u;
        if (j < G.ny - 1 && nat[t + G.nx]) fb |= 8u;
        if (k > 0 && nat[t - nxy]) fb |= 16u;
        if (k < G.nz - 1 && nat[t + nxy]) fb |= 32u;
    }
    in[cell_at(G, i, j, k)] = (unsigned char)fb;
}

// covered cells (mask == 0) of a level-0 mask, accumulated into *out (the caller zeroes it)
__global__ void mask_count_covered_kernel(const unsigned char* __restrict__ mask, long long n, unsigned long long* out)
{
    unsigned long long c = 0;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) c += mask[t] == 0;
    for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
    if ((threadIdx.x & 31) == 0 && c) atomicAdd(out, c);
}

// Self-check (vmg_debug_pad_check): counts the non-zero elements among everything of a padded internal array that is not a
// cell -- the `pad` doubles before and after it and the pad elements of every half row.  The kernels rely on these being
// zero (they stand for the neighbours beyond the domain) and never write them; a stray store shows up here.
__global__ void pad_check_kernel(Geom G, const double* __restrict__ arr, long long pad, unsigned long long* out)
{
    const long long total = 2 * pad + G.plane * G.nz;
    unsigned long long bad = 0;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const long long q = t - pad;                       // index relative to cell 0
        bool is_cell = false;
        if (q >= 0 && q < G.plane * G.nz) {
            const int in_row = (int)(q % G.pitch);
            const int half = in_row / G.hp, m = in_row - half * G.hp;
            is_cell = half == 0 ? m < G.ne : m < G.nx / 2;
        }
        if (!is_cell && arr[q] != 0.0) ++bad;
    }
    for (int o = 16; o > 0; o >>= 1) bad += __shfl_xor_sync(0xffffffffu, bad, o);
    if ((threadIdx.x & 31) == 0 && bad) atomicAdd(out, bad);
}

// public (natural) layout <-> internal layout of one cell array
// mask (may be NULL): covered cells enter as zero (they are identity rows of the masked operator)
// max_out (may be NULL): max |value| stored, so that the solve can tell a zero initial guess (whose residual is btilde itself)
__global__ void to_internal_kernel(Geom G, const double* __restrict__ nat, double* __restrict__ in, const unsigned char* __restrict__ mask,
                                   unsigned long long* max_out = nullptr)
{
    const long long T = (long long)gridDim.x * blockDim.x, t0 = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    double r[kConvElems];
#pragma unroll
    for (int u = 0; u < kConvElems; ++u) {
        const long long t = t0 + u * T;
        r[u] = (t < G.n && !(mask && !mask[t])) ? nat[t] : 0.0;
    }
    double v = 0.0;
    bool nan = false;
#pragma unroll
    for (int u = 0; u < kConvElems; ++u) {
        const long long t = t0 + u * T;
        if (t < G.n) {
            int i, j, k;
            unflatten(G, t, i, j, k);
            in[cell_at(G, i, j, k)] = r[u];
            const double x = fabs(r[u]);
            nan |= x != x;
            v = fmax(v, x);
        }
    }
    if (max_out) {
        if (nan) v = __longlong_as_double(0x7ff8000000000000ll);
        block_max_to_global(v, max_out);
    }
}
__global__ void to_natural_kernel(Geom G, const double* __restrict__ in, double* __restrict__ nat)
{
    const long long T = (long long)gridDim.x * blockDim.x, t0 = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    double r[kConvElems];
#pragma unroll
    for (int u = 0; u < kConvElems; ++u) {
        const long long t = t0 + u * T;
        int i, j, k;
        if (t < G.n) { unflatten(G, t, i, j, k); r[u] = in[cell_at(G, i, j, k)]; }
    }
#pragma unroll
    for (int u = 0; u < kConvElems; ++u) {
        const long long t = t0 + u * T;
        if (t < G.n) nat[t] = r[u];
    }
}

// ------------------------------------------------------------------------------------------------
// Cell masking (reading N4 in DESIGN.md): covered cells are identity rows, a face
// between a valid and a covered cell is an interior boundary of one kind -- Dirichlet with the value the covered cell
// carries, or zero flux.  Realised on the level-0 raw coefficients, so that averaging, stencil build and every solver
// kernel run unchanged: effective a (0 in covered cells), effective b (0 on every face that touches a covered cell),
// an extra diagonal (2 beta b/h^2 per Dirichlet interface face of a valid cell, 1 in a covered cell; averaged to the
// coarse levels like a) and the interface terms of btilde.  All arrays in the public layout.
// ------------------------------------------------------------------------------------------------
struct MaskArgs {
    const unsigned char* mask; const double* cval;      // cval may be NULL (0)
    const double *a, *bx, *by, *bz;                      // the caller's coefficients (may be NULL)
    double *ea, *ebx, *eby, *ebz, *adiag, *mfold;        // effective coefficients, extra diagonal, interface terms
    int nx, ny, nz, three_d, dirichlet;
    double cx, cy, cz;                                   // beta / h^2
};

__global__ void mask_cells_kernel(MaskArgs g)
{
    long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    const long long n = (long long)g.nx * g.ny * g.nz, nxy = (long long)g.nx * g.ny;
    if (t >= n) return;
    int i = (int)(t % g.nx), j = (int)((t / g.nx) % g.ny), k = (int)(t / nxy);
    if (!g.mask[t]) { g.ea[t] = 0.0; g.adiag[t] = 1.0; g.mfold[t] = 0.0; return; }
    g.ea[t] = g.a ? g.a[t] : 0.0;
    double ad = 0.0, mf = 0.0;
    if (g.dirichlet) {
        auto face = [&](bool inside, long long nb, double b, double c) {   // nb: the neighbour cell across the face
            if (!inside || g.mask[nb]) return;
            ad += 2.0 * c * b;
            mf += 2.0 * c * b * (g.cval ? g.cval[nb] : 0.0);
        };
        const long long fx = i + (long long)(g.nx + 1) * (j + (long long)g.ny * k), fy = i + (long long)g.nx * (j + (long long)(g.ny + 1) * k);
        face(i > 0, t - 1, g.bx ? g.bx[fx] : 1.0, g.cx);
        face(i < g.nx - 1, t + 1, g.bx ? g.bx[fx + 1] : 1.0, g.cx);
        face(j > 0, t - g.nx, g.by ? g.by[fy] : 1.0, g.cy);
        face(j < g.ny - 1, t + g.nx, g.by ? g.by[fy + g.nx] : 1.0, g.cy);
        if (g.three_d) {
            face(k > 0, t - nxy, g.bz ? g.bz[t] : 1.0, g.cz);
            face(k < g.nz - 1, t + nxy, g.bz ? g.bz[t + nxy] : 1.0, g.cz);
        }
    }
    g.adiag[t] = ad; g.mfold[t] = mf;
}

// dir: 0 x faces, 1 y faces, 2 z faces: b = 0 on every face that touches a covered cell
__global__ void mask_faces_kernel(MaskArgs g, int dir)
{
    const int ex = g.nx + (dir == 0), ey = g.ny + (dir == 1), ez = g.nz + (dir == 2);
    long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t >= (long long)ex * ey * ez) return;
    int i = (int)(t % ex), j = (int)((t / ex) % ey), k = (int)(t / ((long long)ex * ey));
    const double* b = dir == 0 ? g.bx : dir == 1 ? g.by : g.bz;
    double* eb = dir == 0 ? g.ebx : dir == 1 ? g.eby : g.ebz;
    const int lim = dir == 0 ? g.nx : dir == 1 ? g.ny : g.nz, pos = dir == 0 ? i : dir == 1 ? j : k;
    auto cell = [&](int d) {                             // the cell on the low (d = -1) / high (d = 0) side of the face
        int ci = i + (dir == 0 ? d : 0), cj = j + (dir == 1 ? d : 0), ck = k + (dir == 2 ? d : 0);
        return (long long)ci + (long long)g.nx * (cj + (long long)g.ny * ck);
    };
    bool open = true;
    if (pos > 0) open = open && g.mask[cell(-1)];
    if (pos < lim) open = open && g.mask[cell(0)];
    eb[t] = open ? (b ? b[t] : 1.0) : 0.0;
}

// ------------------------------------------------------------------------------------------------
// The 7-point relaxation / operator in internal form.  All neighbour reads are in-bounds thanks to the
// zero pads and all out-of-domain neighbours carry a zero weight.
// ------------------------------------------------------------------------------------------------
struct LevelView {
    const double *wx, *wy, *wz, *dinv;
    Geom G;
    // constant face weights (b == NULL in vmg_set_coeffs, i.e. b = 1 on every face of every level, and no mask: the
    // Poisson equation PAPER.md:54 Eq. 3 and the Helmholtz equations of photoionisation): the kernels instantiated
    // with CW = true take the six weights from these three numbers and the cell's position instead of loading them,
    // 2 doubles per cell and half-sweep instead of 5.  Same values, same order of operations: bitwise the results
    // of the general kernels on arrays of ones.
    // cw = 2: the same with a cell mask (vmg_set_mask): a face carries beta/h^2 if the cells on both sides are valid and 0
    // otherwise -- exactly the effective coefficients of the masked operator on level 0 (coarser levels of a masked
    // hierarchy have averaged, fractional b and use the arrays).  mk: one byte per cell in the internal layout, bit f =
    // face f open (mask_face_bits_kernel): half a byte per cell and half-sweep instead of 24.
    double cx, cy, cz;
    int cw;
    const unsigned char* mk;
    // batched multi-component launches: nprob problems with identical grids whose arenas lie
    // pstride doubles apart (vmg_create_batch); the launch's blockIdx.z runs over planes x problems, problem-major, and every
    // array of problem kb is the first problem's array shifted by kb * pstride.  0: a single problem.
    long long pstride;
    int nprob;
};

// plane and problem of a batched launch: k = blockIdx.z -> (k % nz, offset of the problem's arrays)
__device__ __forceinline__ long long batch_split(const LevelView& L, int nz, int& k)
{
    if (!L.pstride) return 0;
    const int kb = k / nz;
    k -= kb * nz;
    return (long long)kb * L.pstride;
}

// the six face weights of cell (i, j, k): low x, high x, low y, high y, low z, high z
template <int CW>
__device__ __forceinline__ void face_weights(const LevelView& L, long long c, long long xm, int i, int j, int k, double (&w)[6])
{
    if (CW == 2) {
        const unsigned fb = L.mk[c];     // bit f: face f is open (both cells valid, not a domain face)
        w[0] = (fb & 1u) ? L.cx : 0.0;   w[1] = (fb & 2u) ? L.cx : 0.0;
        w[2] = (fb & 4u) ? L.cy : 0.0;   w[3] = (fb & 8u) ? L.cy : 0.0;
        w[4] = (fb & 16u) ? L.cz : 0.0;  w[5] = (fb & 32u) ? L.cz : 0.0;
    } else if (CW) {
        w[0] = i > 0 ? L.cx : 0.0;  w[1] = i < L.G.nx - 1 ? L.cx : 0.0;
        w[2] = j > 0 ? L.cy : 0.0;  w[3] = j < L.G.ny - 1 ? L.cy : 0.0;
        w[4] = k > 0 ? L.cz : 0.0;  w[5] = k < L.G.nz - 1 ? L.cz : 0.0;
    } else {
        w[0] = L.wx[c];  w[1] = L.wx[xm + 1];
        w[2] = L.wy[c];  w[3] = L.wy[c + L.G.pitch];
        w[4] = L.wz[c];  w[5] = L.wz[c + L.G.plane];
    }
}

// c: the cell; xm: its low-x neighbour (the high-x neighbour is xm + 1: E_m sits between O_{m-1} and O_m, O_m between
// E_m and E_{m+1}).  Same expression, same order, everywhere a relaxation or a residual is evaluated.
__device__ __forceinline__ double nb_sum(const LevelView& L, const double* phi, long long c, long long xm)
{
    double s = L.wx[c] * phi[xm];
    s = fma(L.wx[xm + 1], phi[xm + 1], s);
    s = fma(L.wy[c], phi[c - L.G.pitch], s);
    s = fma(L.wy[c + L.G.pitch], phi[c + L.G.pitch], s);
    s = fma(L.wz[c], phi[c - L.G.plane], s);
    s = fma(L.wz[c + L.G.plane], phi[c + L.G.plane], s);
    return s;
}

// cell and low-x neighbour of pair m, x-parity par, in the row starting at `row`
__device__ __forceinline__ void pair_addr(const Geom& G, long long row, int m, int par, long long& c, long long& xm)
{
    c = row + m + (par ? G.hp : 0);
    xm = row + m + (par ? 0 : G.hp - 1);
}

// S2 (per-colour path). One colour half-sweep: phi_c <- (rhs_c + sum w phi_nb) / D_c for (i+j+k)%2 == colour.
// (m, j, k): the x-pair slot; the kernel derives it from a 3-D grid (pair_launch_dims in vmg_sched.cuh).
// L2 residency: what the NEXT half-sweep (other colour, opposite direction) needs again are the face weights and the
// phi written here; rhs, 1/D and the neighbours' phi are dead after this read, so they are loaded with the streaming
// (evict-first) policy and do not push the weights out of the 126 MB L2.
// KEEP = 1 (option "phi_keep_cells"): the neighbours' phi with the normal policy -- on levels far larger than the L2 the
// evict-first lines are gone before the next row and plane ask for them (512^3: 12 % more DRAM traffic than algorithmic).
template <int CW, int KEEP = 0>
__device__ __forceinline__ void relax_at(const LevelView& L, double* phi, const double* rhs, int colour, int m, int j, int k, long long off = 0)
{
    const Geom& G = L.G;
    int par = (colour + j + k) & 1;
    if (2 * m + par >= G.nx) return;
    long long c, xm;
    pair_addr(G, off + G.plane * k + (long long)G.pitch * j, m, par, c, xm);
    double w[6];
    face_weights<CW>(L, c, xm, 2 * m + par, j, k, w);
    auto ld = [](const double* q) { return KEEP ? *q : __ldcs(q); };
    double s = w[0] * ld(phi + xm);
    s = fma(w[1], ld(phi + xm + 1), s);
    s = fma(w[2], ld(phi + c - G.pitch), s);
    s = fma(w[3], ld(phi + c + G.pitch), s);
    s = fma(w[4], ld(phi + c - G.plane), s);
    s = fma(w[5], ld(phi + c + G.plane), s);
    phi[c] = __ldcs(L.dinv + c) * (__ldcs(rhs + c) + s);
}

// reverse: walk the level from its last plane to its first.  Consecutive half-sweeps alternate direction, so that
// each one starts on the planes the previous one touched last, which are still in the 126 MB L2 (face weights and
// the phi just written are common to both colours).
template <int CW, int KEEP = 0>
__global__ void smooth_colour_kernel(LevelView L, double* __restrict__ phi, const double* __restrict__ rhs, int colour, int reverse)
{
    grid_dependency_wait();
    // grid (x-pair blocks, row blocks, planes), block (x-pairs, rows): no division to find the cell (pair_launch_dims)
    int m = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y, k = blockIdx.z;
    const long long off = batch_split(L, L.G.nz, k);
    if (reverse) { k = L.G.nz - 1 - k; j = gridDim.y * blockDim.y - 1 - j; }
    if (m < L.G.ne && j < L.G.ny) relax_at<CW, KEEP>(L, phi, rhs, colour, m, j, k, off);
}

__device__ __forceinline__ void block_max_to_global(double v, unsigned long long* out);

// S2 + S6 fused (per-colour path): a colour half-sweep that reads the neighbours from phi_in and writes the relaxed cells
// to phi_out (which may be another array), optionally also forming the residual of the cells it relaxes BEFORE relaxing
// them.  A relaxation computes t = rhs_c + sum w phi_nb anyway; the residual of that cell is t - phi_c / (1/D_c): one more
// half double per cell of traffic and a division instead of a kernel of its own over the whole level (S6 "0 (fused)",
// SURVEY.md 8(a)).  Used by the device-side solve loop (vmg_sched.cuh run_solve_loop): the first (red) half-sweep of cycle
// c+1 takes the norm of the iterate after cycle c -- red cells only, reading R12 -- and writes its red cells to the second
// phi array, so that the iterate itself stays untouched if it turns out to be converged; the black half-sweep that follows
// reads its (all red) neighbours from that array and writes into the first one, after which the cycle continues in place.
// Same expressions, same order as relax_at / residual_at: phi and the norms are bitwise those of the separate kernels.
template <int CW, int KEEP, int NORM>
__global__ void smooth_colour_io_kernel(LevelView L, const double* __restrict__ phi_in, double* __restrict__ phi_out,
                                        const double* __restrict__ rhs, int colour, int reverse, unsigned long long* norm_out)
{
    grid_dependency_wait();
    const Geom& G = L.G;
    int m = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y, k = blockIdx.z;
    if (reverse) { k = G.nz - 1 - k; j = gridDim.y * blockDim.y - 1 - j; }
    double mx = 0.0;
    if (m < G.ne && j < G.ny) {
        const int par = (colour + j + k) & 1;
        if (2 * m + par < G.nx) {
            long long c, xm;
            pair_addr(G, G.plane * k + (long long)G.pitch * j, m, par, c, xm);
            double w[6];
            face_weights<CW>(L, c, xm, 2 * m + par, j, k, w);
            auto ld = [](const double* q) { return KEEP ? *q : __ldcs(q); };
            double s = w[0] * ld(phi_in + xm);
            s = fma(w[1], ld(phi_in + xm + 1), s);
            s = fma(w[2], ld(phi_in + c - G.pitch), s);
            s = fma(w[3], ld(phi_in + c + G.pitch), s);
            s = fma(w[4], ld(phi_in + c - G.plane), s);
            s = fma(w[5], ld(phi_in + c + G.plane), s);
            const double di = __ldcs(L.dinv + c), t = __ldcs(rhs + c) + s;
            if (NORM) {
                mx = fabs(t - ld(phi_in + c) / di);
                if (mx != mx) mx = __longlong_as_double(0x7ff8000000000000ll);
            }
            phi_out[c] = di * t;
        }
    }
    if (NORM) block_max_to_global(mx, norm_out);
}

// S7: the exit rules of the solve (C5 of DESIGN.md), on the device, after cycle c's norm has been accumulated:
// st[0] = ||btilde||, [1] = rtol, [2] = max cycles, [3] = cycles done, [4] = slow-cycle counter, [5] = status,
// hist = st + 8.  Sets the WHILE condition of the solve graph and clears the norm accumulator for the next cycle.
__global__ void solve_decide_kernel(cudaGraphConditionalHandle handle, double* st, unsigned long long* norm_bits)
{
    if (threadIdx.x != 0) return;
    const double norm = __longlong_as_double((long long)*norm_bits);
    *norm_bits = 0ull;
    double* hist = st + 8;
    const int c = (int)st[3] + 1;
    const double rtol = st[1], relres = norm / st[0];
    st[3] = (double)c;
    hist[c] = relres;
    unsigned cont = 1u;
    if (relres != relres || relres > 1.7976931348623157e308) { st[5] = -5.0; cont = 0u; }           // VMG_ERR_DIVERGED
    else if (rtol > 0.0) {
        if (relres <= rtol) { st[5] = 0.0; cont = 0u; }                                           // VMG_OK
        else {
            const int slow = hist[c] >= 0.9 * hist[c - 1] ? (int)st[4] + 1 : 0;
            st[4] = (double)slow;
            if (slow >= 3) { st[5] = 2.0; cont = 0u; }                                            // VMG_STALLED
        }
    }
    if (cont && c >= (int)st[2]) cont = 0u;                                                       // VMG_MAXCYCLES (status as initialised)
    cudaGraphSetConditional(handle, cont);
}

// S4 + S2 fused (per-colour path).  The first colour half-sweep after a coarse-grid correction: a relaxation never
// reads the old value of the cell it overwrites, and all six neighbours of a cell of one colour have the other
// colour, so the correction phi += P e (piecewise constant, R9) is applied to the NEIGHBOURS on the fly and never
// stored: the cells of the other colour keep their uncorrected values in memory until the next half-sweep
// overwrites them.  Valid when at least one full sweep follows (nu2 >= 1).  phi_nb + e is the very addition
// prolong_correct_kernel performs, so results are bitwise those of the two separate kernels.
// Cache policy as in relax_at: rhs, 1/D and the neighbours' phi are dead after this read (streaming loads; KEEP = 1: phi with
// the normal policy on levels far larger than the L2); the coarse e is read by eight fine cells and stays cached.
template <int CW, int KEEP = 0>
__device__ __forceinline__ void relax_prolong_one(const LevelView& L, const Geom& CG, double* phi,
                                                  const double* rhs, const double* e, int colour, int sz,
                                                  int m, int j, int k, long long off = 0)
{
    const Geom& G = L.G;
    int par = (colour + j + k) & 1;
    int i = 2 * m + par;
    if (i >= G.nx) return;
    long long c, xm;
    pair_addr(G, off + G.plane * k + (long long)G.pitch * j, m, par, c, xm);
    const int K = sz == 2 ? (k >> 1) : k;
    // In every direction one neighbour has this cell's own coarse parent and the other the adjacent coarse cell (on the
    // low side for an even fine index, on the high side for an odd one): four coarse values, not six.
    const int I = i >> 1;
    long long cP, xP;
    pair_addr(CG, off + CG.plane * K + (long long)CG.pitch * (j >> 1), I >> 1, I & 1, cP, xP);
    const double eP = e[cP];
    const double eX = (i & 1) ? e[xP + 1] : e[xP];                                  // zero pad beyond the x faces: not used there
    const double eY = (j & 1) ? e[cP + CG.pitch] : e[cP - CG.pitch];
    // out-of-domain neighbours carry a zero weight; their (zero-pad or foreign) value is used uncorrected
    auto ld = [](const double* q) { return KEEP ? *q : __ldcs(q); };
    double vxm = ld(phi + xm), vxp = ld(phi + xm + 1), vym = ld(phi + c - G.pitch), vyp = ld(phi + c + G.pitch),
           vzm = ld(phi + c - G.plane), vzp = ld(phi + c + G.plane);
    if (i > 0) vxm += (i & 1) ? eP : eX;
    if (i < G.nx - 1) vxp += (i & 1) ? eX : eP;
    if (j > 0) vym += (j & 1) ? eP : eY;
    if (j < G.ny - 1) vyp += (j & 1) ? eY : eP;
    if (sz == 2) {
        const double eZ = (k & 1) ? e[cP + CG.plane] : e[cP - CG.plane];
        if (k > 0) vzm += (k & 1) ? eP : eZ;
        if (k < G.nz - 1) vzp += (k & 1) ? eZ : eP;
    } else {
        // 2-D: no z coupling (wz = 0), the z-neighbours are pads
    }
    double w[6];
    face_weights<CW>(L, c, xm, i, j, k, w);
    double s = w[0] * vxm;
    s = fma(w[1], vxp, s);
    s = fma(w[2], vym, s);
    s = fma(w[3], vyp, s);
    s = fma(w[4], vzm, s);
    s = fma(w[5], vzp, s);
    phi[c] = __ldcs(L.dinv + c) * (__ldcs(rhs + c) + s);
}

template <int CW, int KEEP = 0>
__global__ void smooth_colour_prolong_kernel(LevelView L, Geom CG, double* __restrict__ phi, const double* __restrict__ rhs,
                                             const double* __restrict__ e, int colour, int sz, int reverse)
{
    grid_dependency_wait();
    int m = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y, k = blockIdx.z;   // pair_launch_dims
    const long long off = batch_split(L, L.G.nz, k);
    if (reverse) { k = L.G.nz - 1 - k; j = gridDim.y * blockDim.y - 1 - j; }
    if (m < L.G.ne && j < L.G.ny) relax_prolong_one<CW, KEEP>(L, CG, phi, rhs, e, colour, sz, m, j, k, off);
}

// r = rhs - A phi, A phi = D phi - sum w phi_nb, D = 1/dinv.
__device__ __forceinline__ double residual_at(const LevelView& L, const double* phi, const double* rhs, long long c, long long xm)
{
    return rhs[c] + nb_sum(L, phi, c, xm) - phi[c] / L.dinv[c];
}

// the same with the cell's position known (CW: constant face weights, see LevelView).  STREAM = 1: phi, rhs and 1/D
// are read with the streaming (evict-first) policy, as in relax_at -- for the norm at the end of a cycle, after which
// the next kernel needs the face weights again and nothing else that is read here.  STREAM = 2: rhs and 1/D only (the
// residual + restriction: phi and the weights are what the up-stroke should still find in L2).
template <int CW, int STREAM = 0>
__device__ __forceinline__ double residual_at(const LevelView& L, const double* phi, const double* rhs, long long c, long long xm,
                                              int i, int j, int k)
{
    if (!CW && !STREAM) return residual_at(L, phi, rhs, c, xm);
    auto ld = [](const double* p) { return STREAM == 1 ? __ldcs(p) : *p; };
    auto ld2 = [](const double* p) { return STREAM ? __ldcs(p) : *p; };
    double w[6];
    face_weights<CW>(L, c, xm, i, j, k, w);
    double s = w[0] * ld(phi + xm);
    s = fma(w[1], ld(phi + xm + 1), s);
    s = fma(w[2], ld(phi + c - L.G.pitch), s);
    s = fma(w[3], ld(phi + c + L.G.pitch), s);
    s = fma(w[4], ld(phi + c - L.G.plane), s);
    s = fma(w[5], ld(phi + c + L.G.plane), s);
    return ld2(rhs + c) + s - ld(phi + c) / ld2(L.dinv + c);
}

// r in the public layout (single-step entry point)
__global__ void residual_kernel(LevelView L, const double* __restrict__ phi, const double* __restrict__ rhs,
                                double* __restrict__ r)
{
    long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t >= L.G.n) return;
    int i, j, k;
    unflatten(L.G, t, i, j, k);
    long long c, xm;
    pair_addr(L.G, L.G.plane * k + (long long)L.G.pitch * j, i >> 1, i & 1, c, xm);
    r[t] = residual_at(L, phi, rhs, c, xm);
}

// S3 (per-colour path). Fused residual + restriction: one thread per coarse cell; also zeroes the coarse phi.
// (Four lanes per coarse cell with a shuffle gather was tried: 70 us instead of 49 us on 256x128x128, the 64-byte
// runs per row coalesce worse than they gain in occupancy.)
// RED = 1: the level was last touched by a black half-sweep (the pre-smoothing of a down-stroke), so the residual of every
// black child is its own rounding error (reading R12 in DESIGN.md: t - fl(fl(dinv t) / dinv), ~2 ulp of D phi) and only the
// four red children are evaluated: 5 doubles per fine cell instead of 7 (all of phi and the weights, half of rhs and 1/D).
// cdinv (may be NULL): 1/D of the coarse level.  The coarse level starts its down-stroke from phi = 0, so its first red
// half-sweep is phi_red = (1/D) (rhs + 0) and touches nothing else: with cdinv the kernel stores that instead of the zero
// (bitwise what smooth_colour_kernel computes from a zero field) and the coarse level skips the launch.
template <int CW, int RED = 0>
__device__ __forceinline__ void restrict_one(const LevelView& L, const Geom& CG, const double* phi,
                                             const double* rhs, double* crhs, double* cphi,
                                             int sz, int I, int J, int K, long long off = 0, const double* cdinv = nullptr)
{
    double s = 0.0;
    for (int r = 0; r < sz; ++r)
        for (int q = 0; q < 2; ++q) {   // the x-pair first, then accumulated (the blocked kernel sums in this order too)
            const int j = 2 * J + q, k = sz * K + r;
            long long row = off + L.G.plane * k + (long long)L.G.pitch * j, ce, xe, co, xo;
            if (RED) {
                const int par = (j + k) & 1;                           // x-parity of the row's red child: (i + j + k) even
                pair_addr(L.G, row, I, par, ce, xe);
                s += residual_at<CW, CW ? 0 : 2>(L, phi, rhs, ce, xe, 2 * I + par, j, k);
            } else {
                pair_addr(L.G, row, I, 0, ce, xe);
                pair_addr(L.G, row, I, 1, co, xo);
                s += residual_at<CW, CW ? 0 : 2>(L, phi, rhs, ce, xe, 2 * I, j, k) + residual_at<CW, CW ? 0 : 2>(L, phi, rhs, co, xo, 2 * I + 1, j, k);   // rhs, 1/D streamed
            }
        }
    const long long cc = off + cell_at(CG, I, J, K);
    const double v = s / (4.0 * sz);
    crhs[cc] = v;
    if (cphi) cphi[cc] = (cdinv && ((I + J + K) & 1) == 0) ? cdinv[cc] * (v + 0.0) : 0.0;   // + 0.0: the sweep's rhs + sum(w * 0)
}

template <int CW>
__global__ void residual_restrict_kernel(LevelView L, Geom CG, const double* __restrict__ phi, const double* __restrict__ rhs,
                                         double* __restrict__ crhs, double* __restrict__ cphi, int sz, int reverse,
                                         const double* __restrict__ cdinv = nullptr)
{
    grid_dependency_wait();
    // grid (coarse x blocks, coarse row blocks, coarse planes), block (coarse x, coarse rows): cell_launch_dims of the coarse level
    int I = blockIdx.x * blockDim.x + threadIdx.x, J = blockIdx.y * blockDim.y + threadIdx.y, K = blockIdx.z;
    const long long off = batch_split(L, CG.nz, K);
    if (reverse) { K = CG.nz - 1 - K; J = gridDim.y * blockDim.y - 1 - J; }
    if (I < CG.nx && J < CG.ny) restrict_one<CW, 0>(L, CG, phi, rhs, crhs, cphi, sz, I, J, K, off, cdinv);
}

// the red children only (restrict_one<CW, 1>).  Latency-bound (ncu: long-scoreboard stalls, 61 % of the warp slots at 34
// registers): with array weights the kernel is held to 32 registers so that 8 CTAs fit an SM.
template <int CW>
__global__ void __launch_bounds__(kThreads, CW == 0 ? 8 : 5)
residual_restrict_red_kernel(LevelView L, Geom CG, const double* __restrict__ phi, const double* __restrict__ rhs,
                             double* __restrict__ crhs, double* __restrict__ cphi, int sz, int reverse,
                             const double* __restrict__ cdinv = nullptr)
{
    grid_dependency_wait();
    int I = blockIdx.x * blockDim.x + threadIdx.x, J = blockIdx.y * blockDim.y + threadIdx.y, K = blockIdx.z;
    const long long off = batch_split(L, CG.nz, K);
    if (reverse) { K = CG.nz - 1 - K; J = gridDim.y * blockDim.y - 1 - J; }
    if (I < CG.nx && J < CG.ny) restrict_one<CW, 1>(L, CG, phi, rhs, crhs, cphi, sz, I, J, K, off, cdinv);
}

// S4 (per-colour path, nu2 = 0 and the single-step entry point). Fused prolongation + correction (piecewise
// constant, R9): phi_f += e_c[i/2, j/2, k/2].
__device__ __forceinline__ void prolong_one(const Geom& G, const Geom& CG, double* phi, const double* e,
                                            int sz, long long t)
{
    int i, j, k;
    unflatten(G, t, i, j, k);
    phi[cell_at(G, i, j, k)] += e[cell_at(CG, i >> 1, j >> 1, sz == 2 ? (k >> 1) : k)];
}

__global__ void prolong_correct_kernel(Geom G, Geom CG, double* __restrict__ phi, const double* __restrict__ e, int sz)
{
    grid_dependency_wait();
    long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t < G.n) prolong_one(G, CG, phi, e, sz, t);
}

// S4, option prolong = 1 (reading R9): cell-centred trilinear prolongation + correction.  Per direction the fine cell
// lies a quarter of a coarse cell from its parent's centre, towards the next coarse cell if its index is odd, towards
// the previous one if even: weights 3/4 (parent), 1/4 (that neighbour), products over the directions (8 coarse values,
// 4 in 2-D).  A neighbour beyond a domain face is a ghost: -e(parent) at a Dirichlet face, +e(parent) at a Neumann
// face.  Same loop order as the oracle's statement of R9 (z, y, x; parent first).
struct ProlongBC { int dirichlet[6]; };

__device__ __forceinline__ double trilinear_value(const int par[3], const int fine[3], const int n[3], int sz, const ProlongBC& bc,
                                                  const double* e, long long (*at)(const void*, int, int, int), const void* geom)
{
    double v = 0.0;
    const int nzs = sz == 2 ? 2 : 1;
    for (int c = 0; c < nzs; ++c)
        for (int b = 0; b < 2; ++b)
            for (int a = 0; a < 2; ++a) {
                const int s[3] = {a, b, c};
                int use[3];
                double sign = 1.0;
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    int idx = s[d] ? par[d] + ((fine[d] & 1) ? 1 : -1) : par[d];
                    if (idx < 0) { idx = par[d]; sign *= bc.dirichlet[2 * d] ? -1.0 : 1.0; }
                    else if (idx >= n[d]) { idx = par[d]; sign *= bc.dirichlet[2 * d + 1] ? -1.0 : 1.0; }
                    use[d] = idx;
                }
                const double w = (a ? 0.25 : 0.75) * (b ? 0.25 : 0.75) * (sz == 2 ? (c ? 0.25 : 0.75) : 1.0);
                v += w * (sign * e[at(geom, use[0], use[1], use[2])]);
            }
    return v;
}

__device__ inline long long at_geom(const void* g, int i, int j, int k) { return cell_at(*(const Geom*)g, i, j, k); }

__device__ __forceinline__ void prolong_trilinear_one(const Geom& G, const Geom& CG, double* phi, const double* e, int sz,
                                                      const ProlongBC& bc, long long t)
{
    int i, j, k;
    unflatten(G, t, i, j, k);
    const int par[3] = {i >> 1, j >> 1, sz == 2 ? (k >> 1) : k}, fine[3] = {i, j, k}, n[3] = {CG.nx, CG.ny, CG.nz};
    phi[cell_at(G, i, j, k)] += trilinear_value(par, fine, n, sz, bc, e, at_geom, &CG);
}

__global__ void prolong_trilinear_kernel(Geom G, Geom CG, double* __restrict__ phi, const double* __restrict__ e, int sz, ProlongBC bc)
{
    grid_dependency_wait();
    long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t < G.n) prolong_trilinear_one(G, CG, phi, e, sz, bc, t);
}

// ------------------------------------------------------------------------------------------------
// S6. Infinity norms: warp shuffle -> block reduce -> one atomicMax on the bit pattern (non-negative
// doubles order like unsigned 64-bit integers; a NaN's pattern is larger than every finite value, so
// it propagates to the host, which tests for it).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void block_max_to_global(double v, unsigned long long* out)
{
    unsigned long long b = (unsigned long long)__double_as_longlong(fabs(v));
    for (int o = 16; o > 0; o >>= 1) {
        unsigned long long other = __shfl_xor_sync(0xffffffffu, b, o);
        b = other > b ? other : b;
    }
    __shared__ unsigned long long warp_max[32];
    const int tid = threadIdx.x + blockDim.x * threadIdx.y;   // blocks are (x, rows) with x a multiple of the warp, or 1-D
    int lane = tid & 31, w = tid >> 5;
    if (lane == 0) warp_max[w] = b;
    __syncthreads();
    if (w == 0) {
        int nw = (blockDim.x * blockDim.y + 31) >> 5;
        b = lane < nw ? warp_max[lane] : 0ull;
        for (int o = 16; o > 0; o >>= 1) {
            unsigned long long other = __shfl_xor_sync(0xffffffffu, b, o);
            b = other > b ? other : b;
        }
        if (lane == 0 && b != 0ull) atomicMax(out, b);
    }
}

// any array of n doubles (an internal array is passed whole: its pad elements are zero)
__global__ void norm_inf_kernel(const double* __restrict__ v, long long n, unsigned long long* out)
{
    double m = 0.0;
    bool nan = false;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
        double x = fabs(v[t]);
        nan |= (x != x);
        m = fmax(m, x);
    }
    if (nan) m = __longlong_as_double(0x7ff8000000000000ll);
    block_max_to_global(m, out);
}

// ||rhs - A phi||_inf accumulated into *out with atomicMax (the caller zeroes it); one cell per thread, both colours or red only
// (as (like two colour half-sweeps in one launch: 13 loads and a division per thread at full occupancy)
template <int CW, int KEEP = 0>   // KEEP = 1: phi with the normal policy (levels far larger than the L2, see relax_at)
// skip_if_zero (may be NULL): a device scalar; when its bits are 0 the kernel does nothing (vmg_solve's initial residual:
// max |phi_0| == 0 means the residual is btilde, which the host then takes from ||btilde||)
__global__ void __launch_bounds__(kThreads, 8) residual_norm_kernel(LevelView L, const double* __restrict__ phi, const double* __restrict__ rhs,
                                     unsigned long long* out, int reverse, const unsigned long long* skip_if_zero = nullptr,
                                     int zslots = 0)
{
    grid_dependency_wait();
    if (skip_if_zero && *skip_if_zero == 0ull) return;   // uniform over the grid
    const Geom& G = L.G;
    // grid (x-pair blocks, row blocks, planes * colours), block (x-pairs, rows): pair_launch_dims, z extended by the colour.
    // zslots > gridDim.z: the z slots are taken gridDim.z apart (the self-skipping launch keeps its grid small: an
    // empty grid of 32768 CTAs still costs 20 us); batched levels are launched with one slot per blockIdx.z
    const int m = blockIdx.x * blockDim.x + threadIdx.x, j0 = blockIdx.y * blockDim.y + threadIdx.y;
    if (zslots <= 0) zslots = (int)gridDim.z;
    double mx = 0.0;
    long long off = 0;
    for (int z = (int)blockIdx.z; z < zslots; z += (int)gridDim.z) {
        int zz = z, j = j0;
        if (L.pstride) {                              // batched: z = (problem, colour, plane), problem-major
            const int span = zslots / L.nprob, kb = zz / span;
            zz -= kb * span;
            off = (long long)kb * L.pstride;
        }
        int k = zz % G.nz;
        const int colour = zz / G.nz;
        if (reverse) { k = G.nz - 1 - k; j = gridDim.y * blockDim.y - 1 - j; }
        if (m < G.ne && j < G.ny) {
            int par = (colour + j + k) & 1;
            if (2 * m + par < G.nx) {
                long long c, xm;
                pair_addr(G, off + G.plane * k + (long long)G.pitch * j, m, par, c, xm);
                double r = fabs(residual_at<CW, CW ? 0 : KEEP ? 2 : 1>(L, phi, rhs, c, xm, 2 * m + par, j, k));   // constant weights: the level fits L2, keep it there
                if (r != r) r = __longlong_as_double(0x7ff8000000000000ll);
                mx = (r > mx || r != r) ? r : mx;
            }
        }
    }
    block_max_to_global(mx, out + off);               // the members' scalars lie the same stride apart (8-byte units)
}

}  // namespace vmg
