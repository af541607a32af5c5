/*
 * oracle/vmg_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU implementation (fp64, triple loops) of the path the CUDA library
 * computes: cell-centred geometric multigrid for
 *
 *        alpha * a * phi  -  beta * div( b grad phi )  =  f        (uniform Cartesian box)
 *
 * the "Helmholtz equation form" every governing equation is cast into (sec. 4): Poisson
 * Eq. 3, implicit diffusion of Eq. 17, photoionisation Eq. 9
 * (PAPER.md:83).  Discretisation: finite volume on Cartesian cells, second-order central diffusive flux,
 * implicit (sec. 3).  The paper names "multigrid" and nothing else; the
 * components are those BASELINE.json:north_star lists, read as SURVEY.md sec. 8(c) C1-C5 / DESIGN.md
 * "Readings".  Nothing here is blocked, fused or reordered beyond those statements.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may load this.
 * It shares no code with paper_2507_08200_b200/csrc and neither includes the other.
 *
 * Parity pins (tests/test_oracle_pins.py): dense LAPACK solve on 8^3 / 16x8x8, manufactured solutions at
 * second order (configs 1, 2), the paper's printed closed form phi = (x^4 - x)/12 (PAPER.md:186-194,
 * Eq. 24-27), exactness for linear phi, symmetry / positive definiteness, constant-vector row sums,
 * axis-permutation invariance, per-cycle contraction < 0.2.  No function here is "parity unpinned".
 *
 * Layout (x fastest): cell arrays idx = i + nx*(j + ny*k); bx (nx+1)*ny*nz, idx = i + (nx+1)*(j + ny*k),
 * face i lies between cells i-1 and i; by nx*(ny+1)*nz, idx = i + nx*(j + (ny+1)*k); bz nx*ny*(nz+1).
 * BC value planes: x faces j + ny*k, y faces i + nx*k, z faces i + nx*j.  nz == 1 selects the 2-D operator.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

enum { XLO = 0, XHI = 1, YLO = 2, YHI = 3, ZLO = 4, ZHI = 5 };
enum { BC_DIRICHLET = 0, BC_NEUMANN = 1 };
enum { O_OK = 0, O_MAXCYCLES = 1, O_STALLED = 2, O_ERR_ARG = -1, O_ERR_SIZE = -2, O_ERR_STATE = -3,
       O_ERR_SINGULAR = -4, O_ERR_DIVERGED = -5 };

typedef struct {
    int nx, ny, nz;
    double hx, hy, hz;
    double *a, *bx, *by, *bz;   /* coefficients of this level (owned) */
    double *phi, *rhs, *res;    /* work arrays of this level (owned) */
    double *adiag;              /* masking: extra diagonal (interface Dirichlet terms, 1 in covered cells); NULL without a mask */
} olevel;

typedef struct ovmg {
    int nlev, three_d;
    olevel *lev;
    double alpha, beta;
    int bctype[6];
    double *bcval[6];           /* level-0 value planes (owned copies; NULL = homogeneous) */
    int have_coeffs, have_bc;
    unsigned char *mask;        /* level 0: 1 = valid, 0 = covered (owned copy); NULL = no mask */
    int mask_kind;              /* BC kind at every covered-valid interface */
    double *cval;               /* Dirichlet value carried by the covered cells (owned copy; NULL = 0) */
    double *mfold;              /* level 0: interface terms of btilde */
    int nu1, nu2, nbottom;
    int prolong;                /* 0: piecewise constant (R9 default), 1: trilinear (R9 option) */
    int symmetric;              /* 1: symmetric V-cycle (post-smoothing and second half of the bottom black->red) */
    int cycles, status;
    double relres;
    double *hist;
    int hist_len;
} ovmg;

static size_t ncell(const olevel *L) { return (size_t)L->nx * L->ny * L->nz; }
static size_t CI(const olevel *L, int i, int j, int k) { return i + (size_t)L->nx * (j + (size_t)L->ny * k); }
static size_t XI(const olevel *L, int i, int j, int k) { return i + (size_t)(L->nx + 1) * (j + (size_t)L->ny * k); }
static size_t YI(const olevel *L, int i, int j, int k) { return i + (size_t)L->nx * (j + (size_t)(L->ny + 1) * k); }
static size_t ZI(const olevel *L, int i, int j, int k) { return i + (size_t)L->nx * (j + (size_t)L->ny * k); }

/* ---------------------------------------------------------------------------------------------
 * C1. The stencil of cell (i,j,k): neighbour weights w[6] (order XLO..ZHI; 0 where the face is a
 * domain boundary) and the diagonal D.  Interior face: w = beta*b_face/h^2 on the diagonal and as
 * the coupling.  Dirichlet boundary face: 2w on the diagonal (value half a cell away), no coupling.
 * Neumann boundary face: nothing.
 * --------------------------------------------------------------------------------------------- */
static void stencil(const ovmg *h, const olevel *L, int i, int j, int k, double w[6], double *D)
{
    double b[6], hh[6];
    int nd = h->three_d ? 6 : 4, f;
    int at_bnd[6];
    b[XLO] = L->bx[XI(L, i, j, k)];     b[XHI] = L->bx[XI(L, i + 1, j, k)];
    b[YLO] = L->by[YI(L, i, j, k)];     b[YHI] = L->by[YI(L, i, j + 1, k)];
    at_bnd[XLO] = (i == 0);             at_bnd[XHI] = (i == L->nx - 1);
    at_bnd[YLO] = (j == 0);             at_bnd[YHI] = (j == L->ny - 1);
    hh[XLO] = hh[XHI] = L->hx;          hh[YLO] = hh[YHI] = L->hy;
    if (h->three_d) {
        b[ZLO] = L->bz[ZI(L, i, j, k)]; b[ZHI] = L->bz[ZI(L, i, j, k + 1)];
        at_bnd[ZLO] = (k == 0);         at_bnd[ZHI] = (k == L->nz - 1);
        hh[ZLO] = hh[ZHI] = L->hz;
    }
    *D = h->alpha * (L->a ? L->a[CI(L, i, j, k)] : 0.0);
    if (L->adiag) *D += L->adiag[CI(L, i, j, k)];
    for (f = 0; f < 6; ++f) w[f] = 0.0;
    for (f = 0; f < nd; ++f) {
        double wf = h->beta * b[f] / (hh[f] * hh[f]);
        if (!at_bnd[f]) { w[f] = wf; *D += wf; }
        else if (h->bctype[f] == BC_DIRICHLET) { *D += 2.0 * wf; }
    }
}

static double nbsum(const olevel *L, const double *phi, int i, int j, int k, const double w[6])
{
    double s = 0.0;
    if (w[XLO] != 0.0) s += w[XLO] * phi[CI(L, i - 1, j, k)];
    if (w[XHI] != 0.0) s += w[XHI] * phi[CI(L, i + 1, j, k)];
    if (w[YLO] != 0.0) s += w[YLO] * phi[CI(L, i, j - 1, k)];
    if (w[YHI] != 0.0) s += w[YHI] * phi[CI(L, i, j + 1, k)];
    if (w[ZLO] != 0.0) s += w[ZLO] * phi[CI(L, i, j, k - 1)];
    if (w[ZHI] != 0.0) s += w[ZHI] * phi[CI(L, i, j, k + 1)];
    return s;
}

/* (A phi)_c = D_c phi_c - sum_interior w phi_nb   (homogeneous-BC operator of level lev) */
static void apply_level(const ovmg *h, int lev, const double *phi, double *out)
{
    const olevel *L = &h->lev[lev];
    int i, j, k;
#pragma omp parallel for collapse(2) private(i)
    for (k = 0; k < L->nz; ++k)
        for (j = 0; j < L->ny; ++j)
            for (i = 0; i < L->nx; ++i) {
                double w[6], D;
                stencil(h, L, i, j, k, w, &D);
                out[CI(L, i, j, k)] = D * phi[CI(L, i, j, k)] - nbsum(L, phi, i, j, k, w);
            }
}

/* r = rhs - A phi */
static void residual_level(const ovmg *h, int lev, const double *phi, const double *rhs, double *r)
{
    const olevel *L = &h->lev[lev];
    int i, j, k;
#pragma omp parallel for collapse(2) private(i)
    for (k = 0; k < L->nz; ++k)
        for (j = 0; j < L->ny; ++j)
            for (i = 0; i < L->nx; ++i) {
                double w[6], D;
                stencil(h, L, i, j, k, w, &D);
                r[CI(L, i, j, k)] = rhs[CI(L, i, j, k)] - (D * phi[CI(L, i, j, k)] - nbsum(L, phi, i, j, k, w));
            }
}

/* C2. One red-black Gauss-Seidel sweep: red = (i+j+k) even first, then black; no over-relaxation.
 * first = 1 runs every sweep black first, then red: the adjoint order, used by the post-smoothing of the symmetric
 * V-cycle that preconditions conjugate gradients (ovmg_solve_pcg). */
static void smooth_level_order(const ovmg *h, int lev, double *phi, const double *rhs, int nsweeps, int first)
{
    const olevel *L = &h->lev[lev];
    int s, c2, colour, i, j, k;
    for (s = 0; s < nsweeps; ++s)
        for (c2 = 0; c2 < 2; ++c2) {
            colour = (first + c2) & 1;
#pragma omp parallel for collapse(2) private(i)
            for (k = 0; k < L->nz; ++k)
                for (j = 0; j < L->ny; ++j)
                    for (i = 0; i < L->nx; ++i) {
                        double w[6], D;
                        if (((i + j + k) & 1) != colour) continue;
                        stencil(h, L, i, j, k, w, &D);
                        phi[CI(L, i, j, k)] = (rhs[CI(L, i, j, k)] + nbsum(L, phi, i, j, k, w)) / D;
                    }
        }
}

static void smooth_level(const ovmg *h, int lev, double *phi, const double *rhs, int nsweeps)
{
    smooth_level_order(h, lev, phi, rhs, nsweeps, 0);
}

/* C3. Restriction: coarse rhs = mean of the 8 (4 in 2-D) children of the fine residual. */
static void restrict_level(const ovmg *h, int lev, const double *rfine, double *rcoarse)
{
    const olevel *F = &h->lev[lev], *C = &h->lev[lev + 1];
    int sz = h->three_d ? 2 : 1, I, J, K, p, q, s;
    for (K = 0; K < C->nz; ++K)
        for (J = 0; J < C->ny; ++J)
            for (I = 0; I < C->nx; ++I) {
                double sum = 0.0;
                for (s = 0; s < sz; ++s)
                    for (q = 0; q < 2; ++q)
                        for (p = 0; p < 2; ++p)
                            sum += rfine[CI(F, 2 * I + p, 2 * J + q, sz * K + s)];
                rcoarse[CI(C, I, J, K)] = sum / (4.0 * sz);
            }
}

/* C3. Prolongation + correction: piecewise constant, phi_f[i,j,k] += e_c[i/2, j/2, k/2] (R9, default).
 *
 * Option prolong = 1 (SURVEY.md sec. 8(c) R9 / DESIGN.md R9): cell-centred trilinear interpolation.  Per direction
 * the fine cell i lies a quarter of a coarse cell from the centre of its parent I = i/2, towards I+1 if i is odd and
 * towards I-1 if i is even: weights 3/4 (parent) and 1/4 (that neighbour); the 3-D weight is the product (8 coarse
 * values; 4 in 2-D).  A neighbour beyond a domain face is a ghost: -e(parent) at a Dirichlet face (the error vanishes
 * on the face, which lies half a coarse cell from the parent's centre), +e(parent) at a Neumann face. */
static double coarse_or_ghost(const ovmg *h, const olevel *C, const double *e, const int idx[3], const int par[3])
{
    /* idx: requested coarse index per direction (may be -1 or n), par: the parent's index (always inside) */
    int n[3], use[3], d;
    double sign = 1.0;
    n[0] = C->nx; n[1] = C->ny; n[2] = C->nz;
    for (d = 0; d < 3; ++d) {
        use[d] = idx[d];
        if (idx[d] < 0)          { use[d] = par[d]; sign *= (h->bctype[2 * d] == BC_DIRICHLET) ? -1.0 : 1.0; }
        else if (idx[d] >= n[d]) { use[d] = par[d]; sign *= (h->bctype[2 * d + 1] == BC_DIRICHLET) ? -1.0 : 1.0; }
    }
    return sign * e[CI(C, use[0], use[1], use[2])];
}

static void prolong_add_level(const ovmg *h, int lev, double *phifine, const double *ecoarse)
{
    const olevel *F = &h->lev[lev], *C = &h->lev[lev + 1];
    int i, j, k;
    if (!h->prolong) {
        for (k = 0; k < F->nz; ++k)
            for (j = 0; j < F->ny; ++j)
                for (i = 0; i < F->nx; ++i)
                    phifine[CI(F, i, j, k)] += ecoarse[CI(C, i / 2, j / 2, h->three_d ? k / 2 : k)];
        return;
    }
    for (k = 0; k < F->nz; ++k)
        for (j = 0; j < F->ny; ++j)
            for (i = 0; i < F->nx; ++i) {
                int par[3], far[3], sx, sy, sz, nzs = h->three_d ? 2 : 1;
                double v = 0.0;
                par[0] = i / 2; par[1] = j / 2; par[2] = h->three_d ? k / 2 : k;
                far[0] = par[0] + ((i & 1) ? 1 : -1);
                far[1] = par[1] + ((j & 1) ? 1 : -1);
                far[2] = par[2] + ((k & 1) ? 1 : -1);
                for (sz = 0; sz < nzs; ++sz)
                    for (sy = 0; sy < 2; ++sy)
                        for (sx = 0; sx < 2; ++sx) {
                            int idx[3];
                            double w = (sx ? 0.25 : 0.75) * (sy ? 0.25 : 0.75) * (h->three_d ? (sz ? 0.25 : 0.75) : 1.0);
                            idx[0] = sx ? far[0] : par[0];
                            idx[1] = sy ? far[1] : par[1];
                            idx[2] = sz ? far[2] : par[2];
                            v += w * coarse_or_ghost(h, C, ecoarse, idx, par);
                        }
                phifine[CI(F, i, j, k)] += v;
            }
}

/* C3 / R10. Coarse coefficients: a = mean of the children; b on a coarse face = mean of the fine
 * faces lying on it (4 in 3-D, 2 in 2-D).  The coarse operator is the re-discretisation C1 with 2h. */
static void average_coeffs(const ovmg *h, int lev)
{
    const olevel *F = &h->lev[lev];
    olevel *C = &h->lev[lev + 1];
    int sz = h->three_d ? 2 : 1, I, J, K, p, q, s;
    for (K = 0; K < C->nz; ++K)
        for (J = 0; J < C->ny; ++J)
            for (I = 0; I < C->nx; ++I) {
                double sum = 0.0;
                for (s = 0; s < sz; ++s) for (q = 0; q < 2; ++q) for (p = 0; p < 2; ++p)
                    sum += F->a[CI(F, 2 * I + p, 2 * J + q, sz * K + s)];
                C->a[CI(C, I, J, K)] = sum / (4.0 * sz);
                if (F->adiag) {   /* masking: the extra diagonal is averaged like a */
                    double sd = 0.0;
                    for (s = 0; s < sz; ++s) for (q = 0; q < 2; ++q) for (p = 0; p < 2; ++p)
                        sd += F->adiag[CI(F, 2 * I + p, 2 * J + q, sz * K + s)];
                    C->adiag[CI(C, I, J, K)] = sd / (4.0 * sz);
                }
            }
    for (K = 0; K < C->nz; ++K)
        for (J = 0; J < C->ny; ++J)
            for (I = 0; I <= C->nx; ++I) {
                double sum = 0.0;
                for (s = 0; s < sz; ++s) for (q = 0; q < 2; ++q)
                    sum += F->bx[XI(F, 2 * I, 2 * J + q, sz * K + s)];
                C->bx[XI(C, I, J, K)] = sum / (2.0 * sz);
            }
    for (K = 0; K < C->nz; ++K)
        for (J = 0; J <= C->ny; ++J)
            for (I = 0; I < C->nx; ++I) {
                double sum = 0.0;
                for (s = 0; s < sz; ++s) for (p = 0; p < 2; ++p)
                    sum += F->by[YI(F, 2 * I + p, 2 * J, sz * K + s)];
                C->by[YI(C, I, J, K)] = sum / (2.0 * sz);
            }
    if (h->three_d)
        for (K = 0; K <= C->nz; ++K)
            for (J = 0; J < C->ny; ++J)
                for (I = 0; I < C->nx; ++I) {
                    double sum = 0.0;
                    for (q = 0; q < 2; ++q) for (p = 0; p < 2; ++p)
                        sum += F->bz[ZI(F, 2 * I + p, 2 * J + q, 2 * K)];
                    C->bz[ZI(C, I, J, K)] = sum / 4.0;
                }
}

/* C1. btilde = f + boundary terms: Dirichlet face with value g adds 2*beta*b*g/h^2; Neumann face with
 * outward-normal derivative q adds beta*b*q/h (R5).  Level 0 only; coarse levels are homogeneous (R4). */
static void fold_bc(const ovmg *h, const double *rhs, double *bt)
{
    const olevel *L = &h->lev[0];
    int i, j, k, f, nd = h->three_d ? 6 : 4;
    for (k = 0; k < L->nz; ++k)
        for (j = 0; j < L->ny; ++j)
            for (i = 0; i < L->nx; ++i) {
                double v = rhs[CI(L, i, j, k)];
                for (f = 0; f < nd; ++f) {
                    double b, hd, g;
                    int on;
                    size_t pl;
                    switch (f) {
                    case XLO: on = (i == 0);          b = L->bx[XI(L, 0, j, k)];      hd = L->hx; pl = j + (size_t)L->ny * k; break;
                    case XHI: on = (i == L->nx - 1);  b = L->bx[XI(L, L->nx, j, k)];  hd = L->hx; pl = j + (size_t)L->ny * k; break;
                    case YLO: on = (j == 0);          b = L->by[YI(L, i, 0, k)];      hd = L->hy; pl = i + (size_t)L->nx * k; break;
                    case YHI: on = (j == L->ny - 1);  b = L->by[YI(L, i, L->ny, k)];  hd = L->hy; pl = i + (size_t)L->nx * k; break;
                    case ZLO: on = (k == 0);          b = L->bz[ZI(L, i, j, 0)];      hd = L->hz; pl = i + (size_t)L->nx * j; break;
                    default:  on = (k == L->nz - 1);  b = L->bz[ZI(L, i, j, L->nz)];  hd = L->hz; pl = i + (size_t)L->nx * j; break;
                    }
                    if (!on || !h->bcval[f]) continue;
                    g = h->bcval[f][pl];
                    if (h->bctype[f] == BC_DIRICHLET) v += 2.0 * h->beta * b * g / (hd * hd);
                    else                              v += h->beta * b * g / hd;
                }
                if (h->mask) v = h->mask[CI(L, i, j, k)] ? v + h->mfold[CI(L, i, j, k)] : 0.0;
                bt[CI(L, i, j, k)] = v;
            }
}

/* C4. V-cycle on level lev: phi (in/out), rhs. */
static void vcycle(ovmg *h, int lev, double *phi, const double *rhs)
{
    olevel *L = &h->lev[lev];
    const int back = h->symmetric ? 1 : 0;          /* colour order of the second half of the cycle */
    if (lev == h->nlev - 1) {                       /* bottom: fixed sweeps from zero (R11) */
        memset(phi, 0, ncell(L) * sizeof(double));
        if (!h->symmetric) smooth_level(h, lev, phi, rhs, h->nbottom);
        else {                                      /* half of them red->black, the other half black->red */
            smooth_level_order(h, lev, phi, rhs, h->nbottom / 2, 0);
            smooth_level_order(h, lev, phi, rhs, h->nbottom - h->nbottom / 2, 1);
        }
        return;
    }
    smooth_level(h, lev, phi, rhs, h->nu1);
    residual_level(h, lev, phi, rhs, L->res);
    restrict_level(h, lev, L->res, h->lev[lev + 1].rhs);
    memset(h->lev[lev + 1].phi, 0, ncell(&h->lev[lev + 1]) * sizeof(double));
    vcycle(h, lev + 1, h->lev[lev + 1].phi, h->lev[lev + 1].rhs);
    prolong_add_level(h, lev, phi, h->lev[lev + 1].phi);
    smooth_level_order(h, lev, phi, rhs, h->nu2, back);
}

static double norm_inf(const double *v, size_t n)
{
    double m = 0.0;
    size_t q;
    for (q = 0; q < n; ++q) {
        double t = fabs(v[q]);
        if (t != t) return t;      /* NaN propagates */
        if (t > m) m = t;
    }
    return m;
}

/* =============================================================================================
 * Exported interface (host pointers).  Mirrors the vmg_* boundary of include/vmg.h in meaning, with an
 * ovmg_ prefix, plus per-step entry points so that tests can compare single kernels.
 * ============================================================================================= */
static void free_level(olevel *L)
{
    free(L->a); free(L->bx); free(L->by); free(L->bz); free(L->phi); free(L->rhs); free(L->res); free(L->adiag);
}

int ovmg_create(ovmg **out, int nx, int ny, int nz, double dx, double dy, double dz)
{
    ovmg *h;
    int n[3], l, nlev = 1, three_d = nz > 1;
    if (!out) return O_ERR_ARG;
    *out = NULL;
    if (nx < 2 || ny < 2 || nz < 1 || !(dx > 0) || !(dy > 0) || (three_d && !(dz > 0))) return O_ERR_SIZE;
    if (three_d && nz < 2) return O_ERR_SIZE;
    /* R11: halve while every active dimension is even and stays >= 2 */
    n[0] = nx; n[1] = ny; n[2] = nz;
    for (;;) {
        int ok = (n[0] % 2 == 0 && n[0] / 2 >= 2 && n[1] % 2 == 0 && n[1] / 2 >= 2);
        if (three_d) ok = ok && (n[2] % 2 == 0 && n[2] / 2 >= 2);
        if (!ok) break;
        n[0] /= 2; n[1] /= 2; if (three_d) n[2] /= 2;
        ++nlev;
    }
    if ((long)n[0] * n[1] * n[2] > 512) return O_ERR_SIZE;   /* fixed-sweep bottom needs a small grid */
    h = (ovmg *)calloc(1, sizeof(ovmg));
    h->lev = (olevel *)calloc(nlev, sizeof(olevel));
    h->nlev = nlev; h->three_d = three_d;
    h->nu1 = 3; h->nu2 = 3; h->nbottom = 32;                 /* R8, R11 */
    h->prolong = 0;                                          /* R9 */
    h->symmetric = 0;
    for (l = 0; l < nlev; ++l) {
        olevel *L = &h->lev[l];
        size_t nc;
        L->nx = nx >> l; L->ny = ny >> l; L->nz = three_d ? nz >> l : 1;
        L->hx = dx * (1 << l); L->hy = dy * (1 << l); L->hz = three_d ? dz * (1 << l) : 1.0;
        nc = ncell(L);
        L->a = (double *)calloc(nc, sizeof(double));
        L->bx = (double *)calloc((size_t)(L->nx + 1) * L->ny * L->nz, sizeof(double));
        L->by = (double *)calloc((size_t)L->nx * (L->ny + 1) * L->nz, sizeof(double));
        L->bz = (double *)calloc((size_t)L->nx * L->ny * (L->nz + 1), sizeof(double));
        L->phi = (double *)calloc(nc, sizeof(double));
        L->rhs = (double *)calloc(nc, sizeof(double));
        L->res = (double *)calloc(nc, sizeof(double));
    }
    for (l = 0; l < 6; ++l) h->bctype[l] = BC_NEUMANN;
    *out = h;
    return O_OK;
}

int ovmg_destroy(ovmg *h)
{
    int l;
    if (!h) return O_ERR_ARG;
    for (l = 0; l < h->nlev; ++l) free_level(&h->lev[l]);
    for (l = 0; l < 6; ++l) free(h->bcval[l]);
    free(h->mask); free(h->cval); free(h->mfold);
    free(h->lev); free(h->hist); free(h);
    return O_OK;
}

/* a == NULL means a = 0; bx,by,bz all NULL means b = 1 (bz ignored in 2-D). */
/* SURVEY.md sec. 8(f) N4 / PAPER.md:136 ("a mask field is set as 1 inside valid plasma regions while it is set as 0 in
 * covered regions. The linear solvers are disabled in covered regions with one-sided numerical schemes enabled at
 * covered-valid interfaces", "directly specifying flux as well as Dirichlet boundary conditions at interior
 * interfaces").  Reading: every face between a valid and a covered cell is an interior boundary of ONE kind --
 * Dirichlet with the value the covered cell carries (an electrode's potential), discretised like a domain face
 * (two-point flux, 2 beta b/h^2 on the diagonal and 2 beta b g/h^2 on the right-hand side), or homogeneous Neumann
 * (zero flux) -- and covered cells are identity rows holding phi = 0.  Realised on the level's coefficients, so that
 * every other routine is unchanged: faces touching a covered cell get b = 0, a = 0 in covered cells, and the extra
 * diagonal `adiag` carries the Dirichlet interface terms (valid cells) and 1 (covered cells); coarse levels average
 * adiag like a (a coarse cell with any valid child stays in the solve, a fully covered one is an identity row). */
static void apply_mask(ovmg *h)
{
    olevel *L = &h->lev[0];
    int i, j, k, f, nd = h->three_d ? 6 : 4;
    for (k = 0; k < L->nz; ++k)
        for (j = 0; j < L->ny; ++j)
            for (i = 0; i < L->nx; ++i) {
                size_t c = CI(L, i, j, k);
                double ad = 0.0, mf = 0.0;
                if (!h->mask[c]) { L->adiag[c] = 1.0; h->mfold[c] = 0.0; continue; }
                for (f = 0; f < nd; ++f) {
                    int ii = i + (f == XHI) - (f == XLO), jj = j + (f == YHI) - (f == YLO), kk = k + (f == ZHI) - (f == ZLO);
                    double b, hd;
                    if (ii < 0 || ii >= L->nx || jj < 0 || jj >= L->ny || kk < 0 || kk >= L->nz) continue;   /* domain face */
                    if (h->mask[CI(L, ii, jj, kk)]) continue;                                                /* valid neighbour */
                    if (h->mask_kind != BC_DIRICHLET) continue;                                              /* zero flux */
                    b = f < 2 ? L->bx[XI(L, i + (f == XHI), j, k)] : f < 4 ? L->by[YI(L, i, j + (f == YHI), k)]
                                                                          : L->bz[ZI(L, i, j, k + (f == ZHI))];
                    hd = f < 2 ? L->hx : f < 4 ? L->hy : L->hz;
                    ad += 2.0 * h->beta * b / (hd * hd);
                    mf += 2.0 * h->beta * b * (h->cval ? h->cval[CI(L, ii, jj, kk)] : 0.0) / (hd * hd);
                }
                L->adiag[c] = ad; h->mfold[c] = mf;
            }
    /* now cut the couplings: b = 0 on every face that touches a covered cell, a = 0 in covered cells */
    for (k = 0; k < L->nz; ++k)
        for (j = 0; j < L->ny; ++j)
            for (i = 0; i < L->nx; ++i) {
                if (h->mask[CI(L, i, j, k)]) continue;
                L->a[CI(L, i, j, k)] = 0.0;
                L->bx[XI(L, i, j, k)] = 0.0; L->bx[XI(L, i + 1, j, k)] = 0.0;
                L->by[YI(L, i, j, k)] = 0.0; L->by[YI(L, i, j + 1, k)] = 0.0;
                if (h->three_d) { L->bz[ZI(L, i, j, k)] = 0.0; L->bz[ZI(L, i, j, k + 1)] = 0.0; }
            }
}

/* mask: nx*ny*nz bytes (1 valid, 0 covered) or NULL to remove the mask; kind: BC_DIRICHLET / BC_NEUMANN at all
 * covered-valid interfaces; cval: cell array with the Dirichlet value of covered cells, or NULL (0).  The coefficients
 * must be set (again) afterwards: ovmg_set_coeffs applies the mask. */
int ovmg_set_mask(ovmg *h, const unsigned char *mask, int kind, const double *cval)
{
    olevel *L;
    int l;
    if (!h || (kind != BC_DIRICHLET && kind != BC_NEUMANN)) return O_ERR_ARG;
    L = &h->lev[0];
    free(h->mask); free(h->cval); free(h->mfold);
    h->mask = NULL; h->cval = NULL; h->mfold = NULL;
    for (l = 0; l < h->nlev; ++l) { free(h->lev[l].adiag); h->lev[l].adiag = NULL; }
    h->have_coeffs = 0;
    if (!mask) return O_OK;
    h->mask = (unsigned char *)malloc(ncell(L));
    memcpy(h->mask, mask, ncell(L));
    h->mask_kind = kind;
    if (cval) { h->cval = (double *)malloc(ncell(L) * sizeof(double)); memcpy(h->cval, cval, ncell(L) * sizeof(double)); }
    h->mfold = (double *)calloc(ncell(L), sizeof(double));
    for (l = 0; l < h->nlev; ++l) h->lev[l].adiag = (double *)calloc(ncell(&h->lev[l]), sizeof(double));
    return O_OK;
}

int ovmg_set_coeffs(ovmg *h, const double *a, const double *bx, const double *by, const double *bz,
                    double alpha, double beta)
{
    olevel *L;
    size_t q, nbx, nby, nbz;
    int l;
    if (!h) return O_ERR_ARG;
    L = &h->lev[0];
    nbx = (size_t)(L->nx + 1) * L->ny * L->nz; nby = (size_t)L->nx * (L->ny + 1) * L->nz;
    nbz = (size_t)L->nx * L->ny * (L->nz + 1);
    if (!bx != !by) return O_ERR_ARG;
    if (h->three_d && (!bx != !bz)) return O_ERR_ARG;
    if (a) memcpy(L->a, a, ncell(L) * sizeof(double)); else memset(L->a, 0, ncell(L) * sizeof(double));
    if (bx) {
        memcpy(L->bx, bx, nbx * sizeof(double));
        memcpy(L->by, by, nby * sizeof(double));
        if (h->three_d) memcpy(L->bz, bz, nbz * sizeof(double));
    } else {
        for (q = 0; q < nbx; ++q) L->bx[q] = 1.0;
        for (q = 0; q < nby; ++q) L->by[q] = 1.0;
        for (q = 0; q < nbz; ++q) L->bz[q] = 1.0;
    }
    h->alpha = a ? alpha : 0.0;
    h->beta = beta;
    if (h->mask) apply_mask(h);
    for (l = 0; l + 1 < h->nlev; ++l) average_coeffs(h, l);
    h->have_coeffs = 1;
    return O_OK;
}

int ovmg_set_bc(ovmg *h, const int *type, const double *const *value)
{
    const olevel *L;
    size_t sizes[6];
    int f;
    if (!h || !type) return O_ERR_ARG;
    L = &h->lev[0];
    sizes[XLO] = sizes[XHI] = (size_t)L->ny * L->nz;
    sizes[YLO] = sizes[YHI] = (size_t)L->nx * L->nz;
    sizes[ZLO] = sizes[ZHI] = (size_t)L->nx * L->ny;
    for (f = 0; f < 6; ++f)
        if (type[f] != BC_DIRICHLET && type[f] != BC_NEUMANN) return O_ERR_ARG;
    for (f = 0; f < 6; ++f) {
        h->bctype[f] = type[f];
        free(h->bcval[f]); h->bcval[f] = NULL;
        if (value && value[f] && (f < 4 || h->three_d)) {
            h->bcval[f] = (double *)malloc(sizes[f] * sizeof(double));
            memcpy(h->bcval[f], value[f], sizes[f] * sizeof(double));
        }
    }
    h->have_bc = 1;
    return O_OK;
}

int ovmg_set_option(ovmg *h, const char *key, double v)
{
    if (!h || !key) return O_ERR_ARG;
    if (!strcmp(key, "nu1")) { if (v < 0) return O_ERR_ARG; h->nu1 = (int)v; return O_OK; }
    if (!strcmp(key, "nu2")) { if (v < 0) return O_ERR_ARG; h->nu2 = (int)v; return O_OK; }
    if (!strcmp(key, "bottom_sweeps")) { if (v < 1) return O_ERR_ARG; h->nbottom = (int)v; return O_OK; }
    if (!strcmp(key, "symmetric")) { if (v != 0.0 && v != 1.0) return O_ERR_ARG; h->symmetric = (int)v; return O_OK; }
    if (!strcmp(key, "prolong")) { if (v != 0.0 && v != 1.0) return O_ERR_ARG; h->prolong = (int)v; return O_OK; }
    return O_ERR_ARG;
}

static void zero_covered(const ovmg *h, double *phi)
{
    size_t c, n = ncell(&h->lev[0]);
    if (h->mask) for (c = 0; c < n; ++c) if (!h->mask[c]) phi[c] = 0.0;
}

static int singular(const ovmg *h)
{
    if (h->mask && h->mask_kind == BC_DIRICHLET) {   /* a covered cell with a Dirichlet interface pins the solution */
        size_t c, n = ncell(&h->lev[0]);
        for (c = 0; c < n; ++c) if (!h->mask[c]) return 0;
    }
    int f, nd = h->three_d ? 6 : 4;
    for (f = 0; f < nd; ++f) if (h->bctype[f] == BC_DIRICHLET) return 0;
    return h->alpha == 0.0;
}

/* C5. Solve: relres = ||btilde - A phi||_inf / ||btilde||_inf (R12), stall rule, status codes. */
int ovmg_solve(ovmg *h, const double *rhs, double *phi, double rtol, int max_vcycles)
{
    olevel *L;
    double nb, *bt;
    int c, slow = 0;
    if (!h || !rhs || !phi || max_vcycles < 0) return O_ERR_ARG;
    if (!h->have_coeffs || !h->have_bc) return O_ERR_STATE;
    if (singular(h)) return O_ERR_SINGULAR;
    L = &h->lev[0];
    bt = L->rhs;
    free(h->hist);
    h->hist = (double *)calloc((size_t)max_vcycles + 1, sizeof(double));
    h->hist_len = 0; h->cycles = 0; h->relres = 0.0;
    zero_covered(h, phi);
    fold_bc(h, rhs, bt);
    nb = norm_inf(bt, ncell(L));
    if (nb == 0.0) {
        memset(phi, 0, ncell(L) * sizeof(double));
        h->hist[0] = 0.0; h->hist_len = 1;
        return h->status = O_OK;
    }
    residual_level(h, 0, phi, bt, L->res);
    h->hist[0] = h->relres = norm_inf(L->res, ncell(L)) / nb;
    h->hist_len = 1;
    if (!(h->relres == h->relres) || isinf(h->relres)) return h->status = O_ERR_DIVERGED;
    if (rtol > 0.0 && h->relres <= rtol) return h->status = O_OK;
    for (c = 1; c <= max_vcycles; ++c) {
        vcycle(h, 0, phi, bt);
        residual_level(h, 0, phi, bt, L->res);
        h->hist[c] = h->relres = norm_inf(L->res, ncell(L)) / nb;
        h->hist_len = c + 1; h->cycles = c;
        if (!(h->relres == h->relres) || isinf(h->relres)) return h->status = O_ERR_DIVERGED;
        if (rtol > 0.0) {
            if (h->relres <= rtol) return h->status = O_OK;
            slow = (h->hist[c] >= 0.9 * h->hist[c - 1]) ? slow + 1 : 0;
            if (slow >= 3) return h->status = O_STALLED;
        }
    }
    return h->status = O_MAXCYCLES;
}

/* conjugate gradients on A phi = btilde, preconditioned by ONE symmetric V-cycle from a zero
 * guess (pre-smoothing red->black, post-smoothing black->red, nu1 = nu2, the bottom's sweeps half and half; R = P^T/8)
 * -- the remedy for the diffusion-dominated high-contrast regime in which plain V-cycles contract slowly (R17) and for
 * which the paper falls back to HYPRE.  Textbook PCG (Hestenes-Stiefel with preconditioner):
 *     r = b - A x;  z = M^-1 r;  p = z;  rho = <r, z>
 *     repeat:  q = A p;  alpha = rho / <p, q>;  x += alpha p;  r -= alpha q;  relres = ||r||_inf / ||b||_inf;
 *              z = M^-1 r;  rho' = <r, z>;  p = z + (rho'/rho) p;  rho = rho'
 * hist[c] is the norm of the recurrence residual after c iterations; exit rules as in ovmg_solve. */
static double dot(const double *u, const double *v, size_t n)
{
    double s = 0.0;
    size_t i;
    for (i = 0; i < n; ++i) s += u[i] * v[i];
    return s;
}

int ovmg_solve_pcg(ovmg *h, const double *rhs, double *phi, double rtol, int max_iter)
{
    olevel *L;
    double nb, rho, *r, *z, *p, *q;
    size_t n, i;
    int c, slow = 0, keep_sym, status = O_MAXCYCLES;
    if (!h || !rhs || !phi || max_iter < 0) return O_ERR_ARG;
    if (!h->have_coeffs || !h->have_bc) return O_ERR_STATE;
    if (singular(h)) return O_ERR_SINGULAR;
    if (h->nu1 != h->nu2) return O_ERR_ARG;          /* the preconditioner must be symmetric */
    L = &h->lev[0];
    n = ncell(L);
    free(h->hist);
    h->hist = (double *)calloc((size_t)max_iter + 1, sizeof(double));
    h->hist_len = 0; h->cycles = 0; h->relres = 0.0;
    r = (double *)malloc(4 * n * sizeof(double));
    if (!r) return O_ERR_ARG;
    z = r + n; p = z + n; q = p + n;
    zero_covered(h, phi);
    fold_bc(h, rhs, q);                               /* q = btilde for a moment */
    nb = norm_inf(q, n);
    if (nb == 0.0) {
        memset(phi, 0, n * sizeof(double));
        h->hist[0] = 0.0; h->hist_len = 1;
        free(r);
        return h->status = O_OK;
    }
    residual_level(h, 0, phi, q, r);                  /* r = btilde - A phi */
    h->hist[0] = h->relres = norm_inf(r, n) / nb;
    h->hist_len = 1;
    if (!(h->relres == h->relres) || isinf(h->relres)) { free(r); return h->status = O_ERR_DIVERGED; }
    if (rtol > 0.0 && h->relres <= rtol) { free(r); return h->status = O_OK; }
    keep_sym = h->symmetric;
    h->symmetric = 1;
    memset(z, 0, n * sizeof(double));
    vcycle(h, 0, z, r);
    memcpy(p, z, n * sizeof(double));
    rho = dot(r, z, n);
    for (c = 1; c <= max_iter; ++c) {
        double alpha, rho2, beta;
        apply_level(h, 0, p, q);
        alpha = rho / dot(p, q, n);
        for (i = 0; i < n; ++i) { phi[i] += alpha * p[i]; r[i] -= alpha * q[i]; }
        h->hist[c] = h->relres = norm_inf(r, n) / nb;
        h->hist_len = c + 1; h->cycles = c;
        if (!(h->relres == h->relres) || isinf(h->relres)) { status = O_ERR_DIVERGED; break; }
        if (rtol > 0.0) {
            if (h->relres <= rtol) { status = O_OK; break; }
            slow = (h->hist[c] >= 0.9 * h->hist[c - 1]) ? slow + 1 : 0;
            if (slow >= 3) { status = O_STALLED; break; }
        }
        if (c == max_iter) break;
        memset(z, 0, n * sizeof(double));
        vcycle(h, 0, z, r);
        rho2 = dot(r, z, n);
        beta = rho2 / rho;
        rho = rho2;
        for (i = 0; i < n; ++i) p[i] = z[i] + beta * p[i];
    }
    h->symmetric = keep_sym;
    free(r);
    return h->status = status;
}

int ovmg_get_info(const ovmg *h, int *cycles, double *relres, double *history)
{
    if (!h) return O_ERR_ARG;
    if (cycles) *cycles = h->cycles;
    if (relres) *relres = h->relres;
    if (history && h->hist) memcpy(history, h->hist, (size_t)h->hist_len * sizeof(double));
    return O_OK;
}

/* ---- per-step entry points for tests (all arrays are caller-owned host arrays of the level's size) ---- */
int ovmg_num_levels(const ovmg *h) { return h ? h->nlev : O_ERR_ARG; }

int ovmg_level_dims(const ovmg *h, int lev, int *dims)
{
    if (!h || lev < 0 || lev >= h->nlev) return O_ERR_ARG;
    dims[0] = h->lev[lev].nx; dims[1] = h->lev[lev].ny; dims[2] = h->lev[lev].nz;
    return O_OK;
}

int ovmg_get_level_coeffs(const ovmg *h, int lev, double *a, double *bx, double *by, double *bz)
{
    const olevel *L;
    if (!h || lev < 0 || lev >= h->nlev) return O_ERR_ARG;
    L = &h->lev[lev];
    if (a) memcpy(a, L->a, ncell(L) * sizeof(double));
    if (bx) memcpy(bx, L->bx, (size_t)(L->nx + 1) * L->ny * L->nz * sizeof(double));
    if (by) memcpy(by, L->by, (size_t)L->nx * (L->ny + 1) * L->nz * sizeof(double));
    if (bz) memcpy(bz, L->bz, (size_t)L->nx * L->ny * (L->nz + 1) * sizeof(double));
    return O_OK;
}

/* masking: the extra diagonal of level `lev` (reading N4: Dirichlet interface terms of valid cells, 1 in covered cells on
 * level 0; averaged like a on the coarse levels).  Accessor only, for the pins of the coarse average. */
int ovmg_get_level_adiag(const ovmg *h, int lev, double *adiag)
{
    const olevel *L;
    if (!h || lev < 0 || lev >= h->nlev || !adiag) return O_ERR_ARG;
    L = &h->lev[lev];
    if (!L->adiag) return O_ERR_ARG;
    memcpy(adiag, L->adiag, ncell(L) * sizeof(double));
    return O_OK;
}

int ovmg_apply(const ovmg *h, int lev, const double *phi, double *out)
{
    if (!h || lev < 0 || lev >= h->nlev || !h->have_coeffs || !h->have_bc) return O_ERR_ARG;
    apply_level(h, lev, phi, out);
    return O_OK;
}

int ovmg_fold_bc(const ovmg *h, const double *rhs, double *btilde)
{
    if (!h || !h->have_coeffs || !h->have_bc) return O_ERR_ARG;
    fold_bc(h, rhs, btilde);
    return O_OK;
}

int ovmg_smooth(const ovmg *h, int lev, double *phi, const double *rhs, int nsweeps)
{
    if (!h || lev < 0 || lev >= h->nlev) return O_ERR_ARG;
    smooth_level(h, lev, phi, rhs, nsweeps);
    return O_OK;
}

int ovmg_residual(const ovmg *h, int lev, const double *phi, const double *rhs, double *r)
{
    if (!h || lev < 0 || lev >= h->nlev) return O_ERR_ARG;
    residual_level(h, lev, phi, rhs, r);
    return O_OK;
}

int ovmg_restrict(const ovmg *h, int lev, const double *rfine, double *rcoarse)
{
    if (!h || lev < 0 || lev + 1 >= h->nlev) return O_ERR_ARG;
    restrict_level(h, lev, rfine, rcoarse);
    return O_OK;
}

int ovmg_prolong_add(const ovmg *h, int lev, double *phifine, const double *ecoarse)
{
    if (!h || lev < 0 || lev + 1 >= h->nlev) return O_ERR_ARG;
    prolong_add_level(h, lev, phifine, ecoarse);
    return O_OK;
}

/* one V-cycle on level 0 with a caller-supplied (already BC-folded) right-hand side */
int ovmg_vcycle(ovmg *h, double *phi, const double *btilde)
{
    if (!h || !h->have_coeffs || !h->have_bc) return O_ERR_ARG;
    vcycle(h, 0, phi, btilde);
    return O_OK;
}
