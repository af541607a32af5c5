/*
 * oracle/amr_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain CPU implementation (fp64, triple loops) of the two-level COMPOSITE solve the CUDA library exports as vmg_amr_*
 * (second half: "then 2-level composite AMR"): the equation of vmg_oracle.c,
 *
 *        alpha * a * phi  -  beta * div( b grad phi )  =  f,
 *
 * on a uniform box (the coarse AMR level, spacing h) of which box-shaped patches of coarse cells [lo, hi) are covered
 * by a fine AMR level of spacing h/2.  The unknowns are the fine cells of the patches and the coarse cells outside them.
 * The paper: "a non-subcycled approach wherein all adaptive mesh refinement (AMR) levels are advanced with the same
 * time-step.  The composite multilevel multigrid solver from within AMReX is used for each of the governing equations"
 * (PAPER.md:157-159), refinement on cell-centred Cartesian blocks.  It says nothing more, so the
 * discretisation at the coarse-fine interface and the cycle are readings (A1-A5):
 *
 *  A1  refinement ratio 2; one or several box patches; each keeps at least one coarse cell between itself and the domain
 *      boundary in every active direction and is at least two coarse cells wide; two patches are at least two coarse cells
 *      apart in some direction (no coarse cell touches two patches, the interpolation of A2 never reads a covered cell).
 *  A2  coarse-fine face: a two-point flux between the fine cell centre and the value g the coarse field takes at the
 *      point of the adjacent coarse cell C that lies opposite it (normal distance hf/2 + h/2 = 1.5 hf), where the coarse
 *      field is interpolated linearly in the tangential directions:
 *            g = phi_C + sum_t s_t (phi_{C+e_t} - phi_{C-e_t}) / 8,      s_t = +1 (-1) if the fine index in t is odd (even)
 *      ((h/4) * central slope).  Flux per unit area b_f (g - phi_f) / (1.5 hf), b_f the FINE face coefficient.
 *  A3  conservation: the coarse cell C takes, through that face, the sum of the fluxes of the fine faces lying on it.
 *  A4  the cycle (correction scheme, no subcycling): composite residual; ONE V-cycle of the plain coarse operator on the
 *      whole coarse box (vmg_oracle.c, C4) for the residual (under the patch: the mean of the children's residuals) from
 *      a zero guess; the correction is added to the coarse cells and, piecewise constant, to the fine cells; nu_f = 6
 *      red-black Gauss-Seidel sweeps on the fine level (the nu1 + nu2 of a V(3,3) cycle, all after the correction) with
 *      the new coarse values in g; the coarse cells under the patch become the means of their children.
 *  A5  relres = max(||r_c||_inf over uncovered coarse cells, ||r_f||_inf) / max(||btilde_c||_inf uncovered, ||f_f||_inf);
 *      exit rules of C5.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu legs may load this.  It shares no code with
 * paper_2507_08200_b200/csrc.  Pins (tests/test_amr_oracle_pins.py): exactness for linear phi at every interface cell
 * (pins the 1/8, the signs and 1.5 hf), conservation (volume-weighted column sums), a face-by-face dense assembly
 * written independently in the test, second-order convergence of a manufactured solution with variable b, convergence
 * of the cycle to the dense solution with contraction < 0.2.  The coarse V-cycle is vmg_oracle.c's (pinned there).
 *
 * Layouts: coarse arrays as in vmg_oracle.c.  Fine arrays, one set per patch: the patch as a box of fx = 2 (hi[0]-lo[0])
 * etc. cells with its own (fx+1)-, (fy+1)-, (fz+1)-face arrays, x fastest.  nz == 1: 2-D (lo[2], hi[2] ignored, fz = 1).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

enum { XLO = 0, XHI = 1, YLO = 2, YHI = 3, ZLO = 4, ZHI = 5 };
enum { BC_DIRICHLET = 0, BC_NEUMANN = 1 };
enum { O_OK = 0, O_MAXCYCLES = 1, O_STALLED = 2, O_ERR_ARG = -1, O_ERR_SIZE = -2, O_ERR_STATE = -3,
       O_ERR_SINGULAR = -4, O_ERR_DIVERGED = -5 };

/* the single-level oracle (vmg_oracle.c), used for the coarse box: BC folding and the correction V-cycle */
typedef struct ovmg ovmg;
int ovmg_create(ovmg **out, int nx, int ny, int nz, double dx, double dy, double dz);
int ovmg_destroy(ovmg *h);
int ovmg_set_coeffs(ovmg *h, const double *a, const double *bx, const double *by, const double *bz, double alpha, double beta);
int ovmg_set_bc(ovmg *h, const int *type, const double *const *value);
int ovmg_set_option(ovmg *h, const char *key, double v);
int ovmg_fold_bc(const ovmg *h, const double *rhs, double *btilde);
int ovmg_vcycle(ovmg *h, double *phi, const double *btilde);

typedef struct {
    int lo[3], hi[3];           /* the patch in coarse cells, [lo, hi) */
    int m[3];                   /* its fine cells: 2 (hi - lo); m[2] = 1 in 2-D */
    double *af, *bf[3];         /* fine coefficients (owned copies; a may be NULL = 0, b NULL = 1) */
} opatch;

typedef struct oamr {
    int n[3];                   /* coarse box */
    double h[3];                /* coarse spacings */
    int three_d, nd;            /* nd = active directions (2 or 3) */
    int np;                     /* patches */
    opatch *p;
    double alpha, beta;
    double *ac, *bc[3];         /* coarse coefficients (owned copies; a may be NULL = 0) */
    int bctype[6];
    ovmg *hc;                   /* the coarse box as a single-level-oracle hierarchy */
    int have_coeffs, have_bc, nu_f;
    int cycles, status, hist_len;
    double relres, *hist;
} oamr;

static size_t ncoarse(const oamr *h) { return (size_t)h->n[0] * h->n[1] * h->n[2]; }
static size_t nfine(const opatch *P) { return (size_t)P->m[0] * P->m[1] * P->m[2]; }
/* cell and face indices; dir = the direction whose face array it is (that array has one more entry along dir) */
static size_t CC(const oamr *h, int i, int j, int k) { return i + (size_t)h->n[0] * (j + (size_t)h->n[1] * k); }
static size_t FC(const opatch *P, int i, int j, int k) { return i + (size_t)P->m[0] * (j + (size_t)P->m[1] * k); }
static size_t face_index(const int *n, int dir, int i, int j, int k)
{
    int ex = n[0] + (dir == 0), ey = n[1] + (dir == 1);
    return i + (size_t)ex * (j + (size_t)ey * k);
}
static size_t face_count(const int *n, int dir)
{
    return (size_t)(n[0] + (dir == 0)) * (n[1] + (dir == 1)) * (n[2] + (dir == 2));
}
static int in_patch(const oamr *h, const opatch *P, int i, int j, int k)
{
    return i >= P->lo[0] && i < P->hi[0] && j >= P->lo[1] && j < P->hi[1] &&
           (!h->three_d || (k >= P->lo[2] && k < P->hi[2]));
}
/* the patch that covers coarse cell (i,j,k), or -1 */
static int covered(const oamr *h, int i, int j, int k)
{
    int q;
    for (q = 0; q < h->np; ++q) if (in_patch(h, &h->p[q], i, j, k)) return q;
    return -1;
}

/* ---------------------------------------------------------------------------------------------
 * A2. The stencil of fine cell (I,J,K) of patch P: w[f] = beta b_f / hf^2 towards a fine neighbour, wcf[f] =
 * beta b_f / (1.5 hf^2) across a patch face (two-point flux over 1.5 hf, divided by the cell width hf), D their sum
 * plus alpha a.  Face order XLO..ZHI.
 * --------------------------------------------------------------------------------------------- */
static void fine_stencil(const oamr *h, const opatch *P, int I, int J, int K, double w[6], double wcf[6], double *D)
{
    int idx[3], f;
    idx[0] = I; idx[1] = J; idx[2] = K;
    *D = h->alpha * (P->af ? P->af[FC(P, I, J, K)] : 0.0);
    for (f = 0; f < 6; ++f) w[f] = wcf[f] = 0.0;
    for (f = 0; f < 2 * h->nd; ++f) {
        int d = f / 2, side = f % 2, p[3];
        double hf = 0.5 * h->h[d], b, wf;
        p[0] = I; p[1] = J; p[2] = K;
        p[d] += side;                                   /* the face on the high side of cell p is face p + 1 */
        b = P->bf[d] ? P->bf[d][face_index(P->m, d, p[0], p[1], p[2])] : 1.0;
        wf = h->beta * b / (hf * hf);
        if ((side == 0 && idx[d] == 0) || (side == 1 && idx[d] == P->m[d] - 1)) { wcf[f] = wf / 1.5; *D += wcf[f]; }
        else { w[f] = wf; *D += wf; }
    }
}

/* A2. g for fine cell (I,J,K) of patch P and its patch face f: the coarse field at the point opposite the fine cell centre */
static double ghost(const oamr *h, const opatch *P, const double *phic, int I, int J, int K, int f)
{
    int d = f / 2, side = f % 2, fi[3], c[3], t;
    double g;
    fi[0] = I; fi[1] = J; fi[2] = K;
    for (t = 0; t < 3; ++t) c[t] = t < h->nd ? P->lo[t] + fi[t] / 2 : 0;
    c[d] += side ? 1 : -1;                              /* the coarse cell across the face */
    g = phic[CC(h, c[0], c[1], c[2])];
    for (t = 0; t < h->nd; ++t) {
        int p[3], q[3];
        double s;
        if (t == d) continue;
        memcpy(p, c, sizeof p); memcpy(q, c, sizeof q);
        p[t] += 1; q[t] -= 1;
        s = (fi[t] % 2) ? 1.0 : -1.0;                   /* the fine centre lies h/4 above (odd) or below (even) C's centre */
        g += s * (phic[CC(h, p[0], p[1], p[2])] - phic[CC(h, q[0], q[1], q[2])]) / 8.0;
    }
    return g;
}

/* sum over the neighbours of fine cell (I,J,K): w phi_nb inside the patch, wcf g across a patch face */
static double fine_nbsum(const oamr *h, const opatch *P, const double *phic, const double *phif, int I, int J, int K,
                         const double w[6], const double wcf[6])
{
    static const int off[6][3] = {{-1, 0, 0}, {1, 0, 0}, {0, -1, 0}, {0, 1, 0}, {0, 0, -1}, {0, 0, 1}};
    double s = 0.0;
    int f;
    for (f = 0; f < 2 * h->nd; ++f) {
        if (w[f] != 0.0) s += w[f] * phif[FC(P, I + off[f][0], J + off[f][1], K + off[f][2])];
        if (wcf[f] != 0.0) s += wcf[f] * ghost(h, P, phic, I, J, K, f);
    }
    return s;
}

/* (A phi)_f = D phi_f - sum w phi_nb - sum wcf g   on every fine cell of patch P */
static void fine_apply(const oamr *h, const opatch *P, const double *phic, const double *phif, double *out)
{
    int I, J, K;
#pragma omp parallel for collapse(2) private(I)
    for (K = 0; K < P->m[2]; ++K)
        for (J = 0; J < P->m[1]; ++J)
            for (I = 0; I < P->m[0]; ++I) {
                double w[6], wcf[6], D;
                fine_stencil(h, P, I, J, K, w, wcf, &D);
                out[FC(P, I, J, K)] = D * phif[FC(P, I, J, K)] - fine_nbsum(h, P, phic, phif, I, J, K, w, wcf);
            }
}

/* A4. red-black Gauss-Seidel on patch P, coarse values fixed: red = (I+J+K) even first (R7; patch-local and
 * global fine indices have the same parity because a patch starts at an even fine index) */
static void fine_smooth(const oamr *h, const opatch *P, const double *phic, double *phif, const double *rhsf, int nsweeps)
{
    int s, colour, I, J, K;
    for (s = 0; s < nsweeps; ++s)
        for (colour = 0; colour < 2; ++colour) {
#pragma omp parallel for collapse(2) private(I)
            for (K = 0; K < P->m[2]; ++K)
                for (J = 0; J < P->m[1]; ++J)
                    for (I = 0; I < P->m[0]; ++I) {
                        double w[6], wcf[6], D;
                        if (((I + J + K) & 1) != colour) continue;
                        fine_stencil(h, P, I, J, K, w, wcf, &D);
                        phif[FC(P, I, J, K)] = (rhsf[FC(P, I, J, K)] + fine_nbsum(h, P, phic, phif, I, J, K, w, wcf)) / D;
                    }
        }
}

/* ---------------------------------------------------------------------------------------------
 * A3. (A phi)_C on the uncovered coarse cells (0 on the covered ones): C1 of vmg_oracle.c with homogeneous boundary
 * values, except across a face shared with a covered cell, through which C takes the fluxes of the fine faces lying
 * on it: sum over them of  beta b_f (g - phi_f) / (1.5 hf) * area_f / volume_C.  phif[q]: the fine field of patch q.
 * --------------------------------------------------------------------------------------------- */
static void coarse_apply(const oamr *h, const double *phic, const double *const *phif, double *out)
{
    int i, j, k;
#pragma omp parallel for collapse(2) private(i)
    for (k = 0; k < h->n[2]; ++k)
        for (j = 0; j < h->n[1]; ++j)
            for (i = 0; i < h->n[0]; ++i) {
                int c[3], f;
                double acc, pc = phic[CC(h, i, j, k)];
                if (covered(h, i, j, k) >= 0) { out[CC(h, i, j, k)] = 0.0; continue; }
                c[0] = i; c[1] = j; c[2] = k;
                acc = h->alpha * (h->ac ? h->ac[CC(h, i, j, k)] : 0.0) * pc;
                for (f = 0; f < 2 * h->nd; ++f) {
                    int d = f / 2, side = f % 2, p[3], q[3], pq;
                    double b, w;
                    memcpy(p, c, sizeof p); memcpy(q, c, sizeof q);
                    p[d] += side;                           /* the face */
                    q[d] += side ? 1 : -1;                  /* the cell across it */
                    b = h->bc[d] ? h->bc[d][face_index(h->n, d, p[0], p[1], p[2])] : 1.0;
                    w = h->beta * b / (h->h[d] * h->h[d]);
                    if (q[d] < 0 || q[d] >= h->n[d]) {      /* domain boundary: Dirichlet value half a cell away (R3) */
                        if (h->bctype[f] == BC_DIRICHLET) acc += 2.0 * w * pc;
                    } else if ((pq = covered(h, q[0], q[1], q[2])) < 0) {
                        acc += w * (pc - phic[CC(h, q[0], q[1], q[2])]);
                    } else {                                /* coarse-fine face of patch pq: the fine faces lying on it */
                        const opatch *P = &h->p[pq];
                        int F[3], t, u, nt = h->nd - 1, tdir[2], ff = 2 * d + (1 - side), fp[3];
                        double hf = 0.5 * h->h[d], area = 1.0, vol = 1.0;
                        for (t = 0, u = 0; t < h->nd; ++t) {
                            vol *= h->h[t];
                            if (t != d) { area *= 0.5 * h->h[t]; tdir[u++] = t; }
                        }
                        for (u = 0; u < (1 << nt); ++u) {
                            double bfine, wp;
                            F[0] = F[1] = F[2] = 0;
                            F[d] = side ? 0 : P->m[d] - 1;
                            for (t = 0; t < nt; ++t) F[tdir[t]] = 2 * (c[tdir[t]] - P->lo[tdir[t]]) + ((u >> t) & 1);
                            memcpy(fp, F, sizeof fp);
                            fp[d] += 1 - side;              /* the fine cell's face towards C */
                            bfine = P->bf[d] ? P->bf[d][face_index(P->m, d, fp[0], fp[1], fp[2])] : 1.0;
                            wp = h->beta * bfine / (1.5 * hf) * area / vol;
                            acc += wp * (ghost(h, P, phic, F[0], F[1], F[2], ff) - phif[pq][FC(P, F[0], F[1], F[2])]);
                        }
                    }
                }
                out[CC(h, i, j, k)] = acc;
            }
}

/* the coarse cells under patch P become the means of their children (A4, last step) */
static void average_down(const oamr *h, const opatch *P, double *phic, const double *phif)
{
    int i, j, k, p, q, s, ns = h->three_d ? 2 : 1;
    for (k = (h->three_d ? P->lo[2] : 0); k < (h->three_d ? P->hi[2] : 1); ++k)
        for (j = P->lo[1]; j < P->hi[1]; ++j)
            for (i = P->lo[0]; i < P->hi[0]; ++i) {
                double sum = 0.0;
                int K0 = h->three_d ? 2 * (k - P->lo[2]) : 0;
                for (s = 0; s < ns; ++s)
                    for (q = 0; q < 2; ++q)
                        for (p = 0; p < 2; ++p)
                            sum += phif[FC(P, 2 * (i - P->lo[0]) + p, 2 * (j - P->lo[1]) + q, K0 + s)];
                phic[CC(h, i, j, k)] = sum / (h->three_d ? 8.0 : 4.0);
            }
}

static double norm_inf(const double *v, size_t n)
{
    double m = 0.0;
    size_t i;
    for (i = 0; i < n; ++i) {
        double x = fabs(v[i]);
        if (!(x == x)) return x;
        if (x > m) m = x;
    }
    return m;
}

static void zero_covered(const oamr *h, double *vc)
{
    int i, j, k;
    for (k = 0; k < h->n[2]; ++k)
        for (j = 0; j < h->n[1]; ++j)
            for (i = 0; i < h->n[0]; ++i)
                if (covered(h, i, j, k) >= 0) vc[CC(h, i, j, k)] = 0.0;
}

/* composite residual: rf[q] = rhsf[q] - A_f on patch q, rc = btc - A_c on the uncovered coarse cells (0 on the covered ones) */
static void composite_residual(const oamr *h, const double *btc, const double *const *rhsf, const double *phic,
                               const double *const *phif, double *rc, double *const *rf)
{
    size_t t, nc = ncoarse(h);
    int q;
    for (q = 0; q < h->np; ++q) {
        size_t nf = nfine(&h->p[q]);
        fine_apply(h, &h->p[q], phic, phif[q], rf[q]);
        for (t = 0; t < nf; ++t) rf[q][t] = rhsf[q][t] - rf[q][t];
    }
    coarse_apply(h, phic, phif, rc);
    for (t = 0; t < nc; ++t) rc[t] = btc[t] - rc[t];
    zero_covered(h, rc);
}

/* ---- the boundary (mirrors vmg_amr_* of include/vmg.h, host pointers).  Patches: lo, hi = npatch triples, flattened;
 * per-patch arrays are passed as arrays of npatch pointers. ---------------------------------------------------- */
int oamr_destroy(oamr *h)
{
    int d, q;
    if (!h) return O_ERR_ARG;
    if (h->hc) ovmg_destroy(h->hc);
    free(h->ac); free(h->hist);
    for (d = 0; d < 3; ++d) free(h->bc[d]);
    for (q = 0; q < h->np; ++q) {
        free(h->p[q].af);
        for (d = 0; d < 3; ++d) free(h->p[q].bf[d]);
    }
    free(h->p);
    free(h);
    return O_OK;
}

int oamr_create(oamr **out, int nx, int ny, int nz, double dx, double dy, double dz, int npatch, const int *lo, const int *hi)
{
    oamr *h;
    int d, q, r, rc;
    if (!out || !lo || !hi || npatch < 1) return O_ERR_ARG;
    h = (oamr *)calloc(1, sizeof(oamr));
    if (!h) return O_ERR_ARG;
    h->n[0] = nx; h->n[1] = ny; h->n[2] = nz;
    h->h[0] = dx; h->h[1] = dy; h->h[2] = dz;
    h->three_d = nz > 1; h->nd = h->three_d ? 3 : 2;
    h->nu_f = 6;
    h->np = npatch;
    h->p = (opatch *)calloc((size_t)npatch, sizeof(opatch));
    for (q = 0; q < npatch; ++q)
        for (d = 0; d < 3; ++d) {
            opatch *P = &h->p[q];
            if (d < h->nd) {
                P->lo[d] = lo[3 * q + d]; P->hi[d] = hi[3 * q + d];
                /* A1: inside the box, one coarse cell away from its boundary, at least two coarse cells wide */
                if (P->lo[d] < 1 || P->hi[d] > h->n[d] - 1 || P->hi[d] - P->lo[d] < 2) { oamr_destroy(h); return O_ERR_SIZE; }
                P->m[d] = 2 * (P->hi[d] - P->lo[d]);
            } else { P->lo[d] = 0; P->hi[d] = 1; P->m[d] = 1; }
        }
    for (q = 0; q < npatch; ++q)                             /* A1: two patches at least two coarse cells apart in some direction */
        for (r = q + 1; r < npatch; ++r) {
            int apart = 0;
            for (d = 0; d < h->nd; ++d)
                if (h->p[r].lo[d] - h->p[q].hi[d] >= 2 || h->p[q].lo[d] - h->p[r].hi[d] >= 2) apart = 1;
            if (!apart) { oamr_destroy(h); return O_ERR_SIZE; }
        }
    rc = ovmg_create(&h->hc, nx, ny, nz, dx, dy, dz);
    if (rc != O_OK) { h->hc = NULL; oamr_destroy(h); return rc; }
    *out = h;
    return O_OK;
}

static double *copy_or_null(const double *src, size_t n)
{
    double *p;
    if (!src) return NULL;
    p = (double *)malloc(n * sizeof(double));
    memcpy(p, src, n * sizeof(double));
    return p;
}

/* coarse coefficients on the whole coarse box (under a patch they define the operator of the correction V-cycle;
 * the caller keeps them consistent with the fine ones), fine coefficients per patch.  NULL a = 0, NULL b = 1
 * (af etc. may be NULL altogether, or hold NULL entries). */
int oamr_set_coeffs(oamr *h, const double *ac, const double *bxc, const double *byc, const double *bzc,
                    const double *const *af, const double *const *bxf, const double *const *byf, const double *const *bzf,
                    double alpha, double beta)
{
    const double *bc[3];
    const double *const *bf[3];
    int d, q, rc;
    if (!h) return O_ERR_ARG;
    bc[0] = bxc; bc[1] = byc; bc[2] = bzc; bf[0] = bxf; bf[1] = byf; bf[2] = bzf;
    free(h->ac);
    h->ac = copy_or_null(ac, ncoarse(h));
    for (d = 0; d < 3; ++d) {
        free(h->bc[d]);
        h->bc[d] = d < h->nd ? copy_or_null(bc[d], face_count(h->n, d)) : NULL;
    }
    for (q = 0; q < h->np; ++q) {
        opatch *P = &h->p[q];
        free(P->af);
        P->af = copy_or_null(af ? af[q] : NULL, nfine(P));
        for (d = 0; d < 3; ++d) {
            free(P->bf[d]);
            P->bf[d] = d < h->nd ? copy_or_null(bf[d] ? bf[d][q] : NULL, face_count(P->m, d)) : NULL;
        }
    }
    h->alpha = alpha; h->beta = beta;
    rc = ovmg_set_coeffs(h->hc, ac, bxc, byc, bzc, alpha, beta);
    if (rc != O_OK) return rc;
    h->have_coeffs = 1;
    return O_OK;
}

/* boundary conditions of the box (the coarse level's; no patch touches the boundary, A1) */
int oamr_set_bc(oamr *h, const int *type, const double *const *value)
{
    int f, rc;
    if (!h || !type) return O_ERR_ARG;
    rc = ovmg_set_bc(h->hc, type, value);
    if (rc != O_OK) return rc;
    for (f = 0; f < 6; ++f) h->bctype[f] = type[f];
    h->have_bc = 1;
    return O_OK;
}

/* "nu_f": fine sweeps per cycle (A4); every other key goes to the coarse hierarchy (nu1, nu2, bottom_sweeps, ...) */
int oamr_set_option(oamr *h, const char *key, double v)
{
    if (!h || !key) return O_ERR_ARG;
    if (!strcmp(key, "nu_f")) { if (v < 1) return O_ERR_ARG; h->nu_f = (int)v; return O_OK; }
    return ovmg_set_option(h->hc, key, v);
}

int oamr_fine_dims(const oamr *h, int patch, int *dims)
{
    if (!h || !dims || patch < 0 || patch >= h->np) return O_ERR_ARG;
    dims[0] = h->p[patch].m[0]; dims[1] = h->p[patch].m[1]; dims[2] = h->p[patch].m[2];
    return O_OK;
}

/* the composite operator with homogeneous boundary values: outc on the uncovered coarse cells (0 under a patch), outf[q] */
int oamr_apply(const oamr *h, const double *phic, const double *const *phif, double *outc, double *const *outf)
{
    int q;
    if (!h || !h->have_coeffs || !h->have_bc || !phic || !phif || !outc || !outf) return O_ERR_ARG;
    for (q = 0; q < h->np; ++q) fine_apply(h, &h->p[q], phic, phif[q], outf[q]);
    coarse_apply(h, phic, phif, outc);
    return O_OK;
}

int oamr_average_down(const oamr *h, double *phic, const double *const *phif)
{
    int q;
    if (!h || !phic || !phif) return O_ERR_ARG;
    for (q = 0; q < h->np; ++q) average_down(h, &h->p[q], phic, phif[q]);
    return O_OK;
}

int oamr_get_info(const oamr *h, int *cycles, double *relres, double *history)
{
    if (!h) return O_ERR_ARG;
    if (cycles) *cycles = h->cycles;
    if (relres) *relres = h->relres;
    if (history && h->hist) memcpy(history, h->hist, (size_t)h->hist_len * sizeof(double));
    return O_OK;
}

/* A4, A5. The composite solve.  rhsc: coarse right-hand side on the whole box (entries under a patch are ignored),
 * rhsf[q]: fine right-hand side of patch q; phic, phif[q]: initial guess in, solution out (phic under a patch: the means
 * of the children).  hist[c] = relres after c cycles. */
int oamr_solve(oamr *h, const double *rhsc, const double *const *rhsf, double *phic, double *const *phif, double rtol, int max_cycles)
{
    size_t t, nc;
    double *btc, *rc, *e, **rf, nb, nrm;
    int c, q, i, j, k, slow = 0, status = O_MAXCYCLES;
    if (!h || !rhsc || !rhsf || !phic || !phif || max_cycles < 0) return O_ERR_ARG;
    if (!h->have_coeffs || !h->have_bc) return O_ERR_STATE;
    nc = ncoarse(h);
    btc = (double *)malloc(nc * sizeof(double)); rc = (double *)malloc(nc * sizeof(double));
    e = (double *)malloc(nc * sizeof(double));
    rf = (double **)malloc((size_t)h->np * sizeof(double *));
    for (q = 0; q < h->np; ++q) rf[q] = (double *)malloc(nfine(&h->p[q]) * sizeof(double));
    free(h->hist);
    h->hist = (double *)calloc((size_t)max_cycles + 1, sizeof(double));
    h->hist_len = 0; h->cycles = 0; h->relres = 0.0;
    ovmg_fold_bc(h->hc, rhsc, btc);                          /* boundary values of the box into the coarse rhs (C1) */
    zero_covered(h, btc);
    nb = norm_inf(btc, nc);
    for (q = 0; q < h->np; ++q) nb = fmax(nb, norm_inf(rhsf[q], nfine(&h->p[q])));
    if (nb == 0.0) {
        memset(phic, 0, nc * sizeof(double));
        for (q = 0; q < h->np; ++q) memset(phif[q], 0, nfine(&h->p[q]) * sizeof(double));
        h->hist[0] = 0.0; h->hist_len = 1;
        status = O_OK;
        goto done;
    }
    for (q = 0; q < h->np; ++q) average_down(h, &h->p[q], phic, phif[q]);
    for (c = 0;; ++c) {
        composite_residual(h, btc, rhsf, phic, (const double *const *)phif, rc, rf);
        nrm = norm_inf(rc, nc);
        for (q = 0; q < h->np; ++q) nrm = fmax(nrm, norm_inf(rf[q], nfine(&h->p[q])));
        h->hist[c] = h->relres = nrm / nb;
        h->hist_len = c + 1; h->cycles = c;
        if (!(h->relres == h->relres) || isinf(h->relres)) { status = O_ERR_DIVERGED; break; }
        if (rtol > 0.0) {
            if (h->relres <= rtol) { status = O_OK; break; }
            if (c > 0) {
                slow = (h->hist[c] >= 0.9 * h->hist[c - 1]) ? slow + 1 : 0;
                if (slow >= 3) { status = O_STALLED; break; }
            }
        }
        if (c == max_cycles) { status = O_MAXCYCLES; break; }
        /* the right-hand side of the coarse correction: the coarse residual, under a patch the mean of the children's */
        for (q = 0; q < h->np; ++q) average_down(h, &h->p[q], rc, rf[q]);
        memset(e, 0, nc * sizeof(double));
        ovmg_vcycle(h->hc, e, rc);
        for (t = 0; t < nc; ++t) phic[t] += e[t];
        for (q = 0; q < h->np; ++q) {
            const opatch *P = &h->p[q];
            for (k = 0; k < P->m[2]; ++k)
                for (j = 0; j < P->m[1]; ++j)
                    for (i = 0; i < P->m[0]; ++i)
                        phif[q][FC(P, i, j, k)] += e[CC(h, P->lo[0] + i / 2, P->lo[1] + j / 2, h->three_d ? P->lo[2] + k / 2 : 0)];
        }
        for (q = 0; q < h->np; ++q) fine_smooth(h, &h->p[q], phic, phif[q], rhsf[q], h->nu_f);
        for (q = 0; q < h->np; ++q) average_down(h, &h->p[q], phic, phif[q]);
    }
done:
    for (q = 0; q < h->np; ++q) free(rf[q]);
    free(rf); free(btc); free(rc); free(e);
    return h->status = status;
}
