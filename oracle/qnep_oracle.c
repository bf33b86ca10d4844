/*
 * qnep_oracle.c -- fp64 CPU ORACLE for the per-step qNEP force evaluation of
 * arXiv 2601.19034.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, the smoke check
 * in __graft_entry__.py and bench.py's cpu_baseline / --impl reference legs may
 * call it.  It shares no code, header, table or constant generator with the
 * CUDA path in paper_2601_19034_b200/; the CUDA path never calls it.
 *
 * It is the plain definition evaluated slowly, in the paper's order and
 * notation; `omp parallel for` over atoms (or k-vectors / mesh lines) is the
 * only concession to run time.  Nothing is blocked, fused or reordered.
 *
 * Passages followed (PAPER.md line : equation), and the DESIGN.md readings
 * where the extracted text is garbled or silent:
 *   neighbours        :91, :138 Eq. 13        all images (j, s), 0 < |r_j+s-r_i| < r_c
 *   descriptors       :56 (-> NEP refs)       reading S1-S3 (Chebyshev radial basis, smooth
 *                                             cutoff, Legendre double sum for the angular part)
 *   NN                :41-45 Eq. 1, :58-60    minus biases; second output node = q_i; S4, S5
 *   neutralisation    :255-262 Eq. 33         reading G3
 *   U^r, U^k, U^s     :85-118 Eq. 6-10        reading G1 (erfc(alpha r), k != 0)
 *   forces / virial   :124-199 Eq. 11-23      dynamic-charge terms folded (:140), reading S6;
 *                                             per-atom virial: Eq. 12, Eq. 20 (real part, G4), Eq. 39
 *   BEC               :205-227 Eq. 24-28      reading S12
 *   field response    :229-237 Eq. 29-30      F^ext = E.Z, Pdot = sum_i Z_i v_i (orc_response)
 *   PPPM              :266-304 Eq. 34-38      readings G2 (Eq. 36), S10 (W, P = 5), S11 (FFT)
 *   4-/5-body terms   :39 (NEP4 -> NEP refs)  reading Z2: cubic invariant of the l = 2 moments, square of the l = 1 invariant
 *   ZBL core          :39 (NEP4 -> NEP refs)  reading Z1: universal ZBL pair repulsion with a cosine switch (optional,
 *                                             orc_set_zbl)
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): NaCl Madelung constant,
 * Ewald vs brute-force image sum, alpha independence, U = 1/2 sum q phi + U^s,
 * finite-difference forces and finite-strain virials, PPPM adjointness identity,
 * PPPM -> Ewald convergence, invariants, Legendre double sum vs spherical
 * harmonics (scipy), FFT vs numpy, B-spline vs its convolution definition,
 * alias-sum denominator vs brute force, BEC vs finite differences of q and of the cluster
 * polarization P = sum q~_i r_i (Eq. 26-28), Eq. 1 evaluated by hand (bias signs, per-type blocks),
 * Eq. 29-30 vs the point-charge limit (F = q E, Pdot = sum q v), the power identity, a case evaluated by
 * hand and finite differences of E.P and of P(t) (index order of Z); ZBL vs the bare-Coulomb limit r -> 0, the switch
 * end points, finite-difference forces and finite-strain virials.
 * No function here is "parity unpinned".
 *
 * Units: Angstrom, eV, elementary charge.  K = 1/(4 pi eps0) (reading S9).
 * Layout: positions and forces are component-major [3][N]; box[9] rows are the
 * cell vectors a, b, c.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_K_COULOMB 14.3996454784 /* eV*A/e^2, reading S9 */
#define ORC_PI 3.14159265358979323846

typedef struct {
    int32_t n_types, n_max_r, n_max_a, l_max, basis_r, basis_a, n_neurons;
    double rc_r, rc_a;
    int32_t mode;              /* 1: U^r+U^k+U^s (Eq. 3); 2: U^k only (Eq. 5) */
    double sqrt_eps_inf, q_total;
    int32_t l_max_4b, l_max_5b; /* NEP4 higher-body angular terms (reading Z2): 2 / 1 to switch them on, 0 = off */
} orc_model;

typedef struct {
    int32_t method;            /* 0 none, 1 Ewald, 2 PPPM */
    double alpha;              /* <= 0 -> pi / rc_r (:91) */
    int32_t ewald_nmax2;       /* > 0: keep integer n.n <= nmax2 (S7); <= 0: |k| <= 2 pi alpha (:110) */
    int32_t grid[3];
    int32_t order;             /* P; only 5 is implemented (:280) */
} orc_es;

/* optional per-stage outputs of orc_compute (any pointer may be NULL) */
typedef struct {
    double *D;       /* [N][n_desc]  unscaled descriptors                           */
    double *U_i;     /* [N]          site energies (Eq. 1)                          */
    double *q_raw;   /* [N]          charges before Eq. 33                          */
    double *phi;     /* [N]          dU^ES/dq_i before the S6 mean subtraction      */
    double *Fp;      /* [N][n_desc]  dU_i/dD + phi_eff dq_i/dD                      */
    double *rho;     /* [Nx][Ny][Nz] PPPM charge mesh (z fastest)                   */
    double *F_es;    /* [3][N]       static electrostatic force only                */
} orc_debug;

void orc_zbl_pair(double r, double Zi, double Zj, double r1, double r2, double *u, double *du);
/* optional ZBL core (reading Z1), switched on for the calls that follow by orc_set_zbl */
#define ORC_MAX_TYPES 8
static struct { int on; double r1, r2; double Z[ORC_MAX_TYPES]; } g_zbl = {0, 0.0, 0.0, {0}};

void orc_set_zbl(int on, double r_inner, double r_outer, const double *Z, int n_types)
{
    g_zbl.on = on && r_outer > 0.0;
    g_zbl.r1 = r_inner;
    g_zbl.r2 = r_outer;
    for (int t = 0; t < ORC_MAX_TYPES; ++t) g_zbl.Z[t] = (Z && t < n_types) ? Z[t] : 0.0;
}

/* ------------------------------------------------------------------------- */
/* small helpers                                                              */
/* ------------------------------------------------------------------------- */
int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

static double det3(const double *h)
{
    return h[0] * (h[4] * h[8] - h[5] * h[7]) - h[1] * (h[3] * h[8] - h[5] * h[6]) +
           h[2] * (h[3] * h[7] - h[4] * h[6]);
}

/* inverse of the 3x3 matrix whose ROWS are a, b, c;  inv columns are the reciprocal
 * vectors / 2 pi:  frac = r . inv  (row vector times matrix). */
static void inv3(const double *h, double *inv)
{
    double d = det3(h);
    inv[0] = (h[4] * h[8] - h[5] * h[7]) / d;
    inv[1] = (h[2] * h[7] - h[1] * h[8]) / d;
    inv[2] = (h[1] * h[5] - h[2] * h[4]) / d;
    inv[3] = (h[5] * h[6] - h[3] * h[8]) / d;
    inv[4] = (h[0] * h[8] - h[2] * h[6]) / d;
    inv[5] = (h[2] * h[3] - h[0] * h[5]) / d;
    inv[6] = (h[3] * h[7] - h[4] * h[6]) / d;
    inv[7] = (h[1] * h[6] - h[0] * h[7]) / d;
    inv[8] = (h[0] * h[4] - h[1] * h[3]) / d;
}

/* wrap positions into the cell; out is [3][N] */
static void wrap_positions(int64_t n, const double *pos, const double *box, double *out)
{
    double inv[9];
    inv3(box, inv);
    for (int64_t i = 0; i < n; ++i) {
        double r[3] = {pos[i], pos[n + i], pos[2 * n + i]};
        double f[3];
        for (int a = 0; a < 3; ++a) {
            f[a] = r[0] * inv[0 * 3 + a] + r[1] * inv[1 * 3 + a] + r[2] * inv[2 * 3 + a];
            f[a] -= floor(f[a]);
            if (f[a] >= 1.0) f[a] = 0.0;
        }
        for (int a = 0; a < 3; ++a)
            out[a * n + i] = f[0] * box[0 * 3 + a] + f[1] * box[1 * 3 + a] + f[2] * box[2 * 3 + a];
    }
}

/* perpendicular heights of the cell along a, b, c */
static void cell_heights(const double *box, double *hgt)
{
    double vol = fabs(det3(box));
    const double *a = box, *b = box + 3, *c = box + 6;
    double bc[3] = {b[1] * c[2] - b[2] * c[1], b[2] * c[0] - b[0] * c[2], b[0] * c[1] - b[1] * c[0]};
    double ca[3] = {c[1] * a[2] - c[2] * a[1], c[2] * a[0] - c[0] * a[2], c[0] * a[1] - c[1] * a[0]};
    double ab[3] = {a[1] * b[2] - a[2] * b[1], a[2] * b[0] - a[0] * b[2], a[0] * b[1] - a[1] * b[0]};
    hgt[0] = vol / sqrt(bc[0] * bc[0] + bc[1] * bc[1] + bc[2] * bc[2]);
    hgt[1] = vol / sqrt(ca[0] * ca[0] + ca[1] * ca[1] + ca[2] * ca[2]);
    hgt[2] = vol / sqrt(ab[0] * ab[0] + ab[1] * ab[1] + ab[2] * ab[2]);
}

/* ------------------------------------------------------------------------- */
/* neighbours (:91, Eq. 13): all (j, s) with 0 < |r_j + s - r_i| < rc         */
/* ------------------------------------------------------------------------- */
typedef struct {
    int64_t n;
    int64_t *start;    /* [n+1] */
    int32_t *j;        /* [start[n]] */
    double *d;         /* [start[n]][4] : r_ij (x, y, z) and |r_ij| */
} orc_nlist;

static void nlist_free(orc_nlist *nl)
{
    free(nl->start);
    free(nl->j);
    free(nl->d);
    memset(nl, 0, sizeof(*nl));
}

/* visit every image neighbour of atom i by brute force; cb==0 counts only */
static int64_t visit_brute(int64_t n, const double *w, const double *box, const int *m, double rc,
                           int64_t i, int32_t *oj, double *od)
{
    int64_t cnt = 0;
    double rc2 = rc * rc;
    for (int64_t j = 0; j < n; ++j)
        for (int s0 = -m[0]; s0 <= m[0]; ++s0)
            for (int s1 = -m[1]; s1 <= m[1]; ++s1)
                for (int s2 = -m[2]; s2 <= m[2]; ++s2) {
                    double d[3];
                    for (int a = 0; a < 3; ++a)
                        d[a] = w[a * n + j] + s0 * box[a] + s1 * box[3 + a] + s2 * box[6 + a] - w[a * n + i];
                    double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
                    if (r2 < rc2 && r2 > 0.0) {
                        if (oj) {
                            oj[cnt] = (int32_t)j;
                            od[4 * cnt + 0] = d[0];
                            od[4 * cnt + 1] = d[1];
                            od[4 * cnt + 2] = d[2];
                            od[4 * cnt + 3] = sqrt(r2);
                        }
                        ++cnt;
                    }
                }
    return cnt;
}

/* binned search (same neighbour set as brute force; pinned by a test) */
typedef struct {
    int nb[3];
    int64_t *bin_start; /* [nbins+1] */
    int32_t *bin_atoms;
    int32_t *atom_bin;  /* [n][3] */
} orc_bins;

static int64_t visit_bins(int64_t n, const double *w, const double *box, const orc_bins *B, double rc,
                          int64_t i, int32_t *oj, double *od)
{
    int64_t cnt = 0;
    double rc2 = rc * rc;
    const int *nb = B->nb;
    for (int d0 = -1; d0 <= 1; ++d0)
        for (int d1 = -1; d1 <= 1; ++d1)
            for (int d2 = -1; d2 <= 1; ++d2) {
                int c[3] = {B->atom_bin[3 * i] + d0, B->atom_bin[3 * i + 1] + d1, B->atom_bin[3 * i + 2] + d2};
                int s[3];
                for (int a = 0; a < 3; ++a) {
                    s[a] = 0;
                    if (c[a] < 0) { c[a] += nb[a]; s[a] = -1; }
                    else if (c[a] >= nb[a]) { c[a] -= nb[a]; s[a] = 1; }
                }
                int64_t bin = ((int64_t)c[0] * nb[1] + c[1]) * nb[2] + c[2];
                for (int64_t p = B->bin_start[bin]; p < B->bin_start[bin + 1]; ++p) {
                    int64_t j = B->bin_atoms[p];
                    double d[3];
                    for (int a = 0; a < 3; ++a)
                        d[a] = w[a * n + j] + s[0] * box[a] + s[1] * box[3 + a] + s[2] * box[6 + a] - w[a * n + i];
                    double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
                    if (r2 < rc2 && r2 > 0.0) {
                        if (oj) {
                            oj[cnt] = (int32_t)j;
                            od[4 * cnt + 0] = d[0];
                            od[4 * cnt + 1] = d[1];
                            od[4 * cnt + 2] = d[2];
                            od[4 * cnt + 3] = sqrt(r2);
                        }
                        ++cnt;
                    }
                }
            }
    return cnt;
}

/* use_bins: 0 brute force, 1 bins if the cell allows (>= 3 bins per axis), else brute force */
static int build_nlist(int64_t n, const double *w, const double *box, double rc, int use_bins, orc_nlist *nl)
{
    double hgt[3];
    int m[3];
    cell_heights(box, hgt);
    for (int a = 0; a < 3; ++a) m[a] = (int)ceil(rc / hgt[a]);
    orc_bins B;
    memset(&B, 0, sizeof(B));
    int bins_ok = use_bins;
    for (int a = 0; a < 3; ++a) {
        B.nb[a] = (int)floor(hgt[a] / rc);
        if (B.nb[a] < 3) bins_ok = 0;
    }
    if (bins_ok) {
        double inv[9];
        inv3(box, inv);
        int64_t nbins = (int64_t)B.nb[0] * B.nb[1] * B.nb[2];
        B.bin_start = (int64_t *)calloc((size_t)(nbins > 0 ? nbins : 1) + 1, sizeof(int64_t));
        B.bin_atoms = (int32_t *)malloc(sizeof(int32_t) * (n > 0 ? n : 1));
        B.atom_bin = (int32_t *)malloc(sizeof(int32_t) * 3 * (n > 0 ? n : 1));
        int64_t *abin = (int64_t *)malloc(sizeof(int64_t) * (n > 0 ? n : 1));
        for (int64_t i = 0; i < n; ++i) {
            int c[3];
            for (int a = 0; a < 3; ++a) {
                double f = w[i] * inv[a] + w[n + i] * inv[3 + a] + w[2 * n + i] * inv[6 + a];
                c[a] = (int)floor(f * B.nb[a]);
                if (c[a] < 0) c[a] = 0;
                if (c[a] >= B.nb[a]) c[a] = B.nb[a] - 1;
                B.atom_bin[3 * i + a] = c[a];
            }
            abin[i] = ((int64_t)c[0] * B.nb[1] + c[1]) * B.nb[2] + c[2];
            B.bin_start[abin[i] + 1]++;
        }
        for (int64_t b = 0; b < nbins; ++b) B.bin_start[b + 1] += B.bin_start[b];
        int64_t *fill = (int64_t *)calloc((size_t)(nbins > 0 ? nbins : 1), sizeof(int64_t));
        for (int64_t i = 0; i < n; ++i) B.bin_atoms[B.bin_start[abin[i]] + fill[abin[i]]++] = (int32_t)i;
        free(fill);
        free(abin);
    }
    nl->n = n;
    nl->start = (int64_t *)calloc(n + 1, sizeof(int64_t));
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i)
        nl->start[i + 1] = bins_ok ? visit_bins(n, w, box, &B, rc, i, 0, 0) : visit_brute(n, w, box, m, rc, i, 0, 0);
    for (int64_t i = 0; i < n; ++i) nl->start[i + 1] += nl->start[i];
    int64_t tot = nl->start[n];
    nl->j = (int32_t *)malloc(sizeof(int32_t) * (tot > 0 ? tot : 1));
    nl->d = (double *)malloc(sizeof(double) * 4 * (tot > 0 ? tot : 1));
    if (!nl->j || !nl->d) return -1;
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
        int32_t *oj = nl->j + nl->start[i];
        double *od = nl->d + 4 * nl->start[i];
        if (bins_ok) visit_bins(n, w, box, &B, rc, i, oj, od);
        else visit_brute(n, w, box, m, rc, i, oj, od);
    }
    free(B.bin_start);
    free(B.bin_atoms);
    free(B.atom_bin);
    return 0;
}

/* exported for the neighbour-set pin: counts[i] and, if cap > 0, the first `cap` (j, rx, ry, rz, r)
 * of every atom, sorted by the caller. */
int orc_neighbors(int64_t n, const double *pos, const double *box, double rc, int use_bins,
                  int64_t *counts, int64_t cap, int32_t *out_j, double *out_d)
{
    double *w = (double *)malloc(sizeof(double) * 3 * (n > 0 ? n : 1));
    wrap_positions(n, pos, box, w);
    orc_nlist nl;
    if (build_nlist(n, w, box, rc, use_bins, &nl)) { free(w); return -1; }
    for (int64_t i = 0; i < n; ++i) {
        int64_t c = nl.start[i + 1] - nl.start[i];
        counts[i] = c;
        for (int64_t p = 0; p < c && p < cap; ++p) {
            out_j[i * cap + p] = nl.j[nl.start[i] + p];
            for (int a = 0; a < 4; ++a) out_d[(i * cap + p) * 4 + a] = nl.d[4 * (nl.start[i] + p) + a];
        }
    }
    nlist_free(&nl);
    free(w);
    return 0;
}

/* ------------------------------------------------------------------------- */
/* descriptors (:56; reading S1-S3)                                           */
/* ------------------------------------------------------------------------- */
/* f_k(r) = 1/2 [T_k(x) + 1] f_c(r),  x = 2 (r/rc - 1)^2 - 1,  f_c = 1/2 [1 + cos(pi r / rc)],  k = 0..nbas */
static void radial_basis(double r, double rc, int nbas, double *f, double *df)
{
    if (r >= rc) {
        for (int k = 0; k <= nbas; ++k) f[k] = df[k] = 0.0;
        return;
    }
    double fc = 0.5 * (1.0 + cos(ORC_PI * r / rc));
    double dfc = -0.5 * ORC_PI / rc * sin(ORC_PI * r / rc);
    double x = 2.0 * (r / rc - 1.0) * (r / rc - 1.0) - 1.0;
    double dx = 4.0 * (r / rc - 1.0) / rc;
    double Tm = 1.0, T = x, dTm = 0.0, dT = 1.0; /* T_0, T_1 and derivatives wrt x */
    for (int k = 0; k <= nbas; ++k) {
        double Tk, dTk;
        if (k == 0) { Tk = 1.0; dTk = 0.0; }
        else if (k == 1) { Tk = x; dTk = 1.0; }
        else {
            Tk = 2.0 * x * T - Tm;
            dTk = 2.0 * T + 2.0 * x * dT - dTm;
            Tm = T; dTm = dT; T = Tk; dT = dTk;
        }
        f[k] = 0.5 * (Tk + 1.0) * fc;
        df[k] = 0.5 * dTk * dx * fc + 0.5 * (Tk + 1.0) * dfc;
    }
}

/* g_n(r) = sum_k c^{ti tj}_{nk} f_k(r) */
static void g_functions(const double *c, int nT, int ti, int tj, int nn, int nbas, const double *f,
                        const double *df, double *g, double *dg)
{
    const double *cc = c + ((size_t)(ti * nT + tj) * nn) * (nbas + 1);
    for (int n = 0; n < nn; ++n) {
        double s = 0.0, ds = 0.0;
        for (int k = 0; k <= nbas; ++k) {
            s += cc[n * (nbas + 1) + k] * f[k];
            ds += cc[n * (nbas + 1) + k] * df[k];
        }
        g[n] = s;
        dg[n] = ds;
    }
}

/* Legendre P_l(c) and dP_l/dc, l = 0..lmax */
static void legendre(double c, int lmax, double *P, double *dP)
{
    P[0] = 1.0; dP[0] = 0.0;
    if (lmax >= 1) { P[1] = c; dP[1] = 1.0; }
    for (int l = 1; l < lmax; ++l) {
        P[l + 1] = ((2 * l + 1) * c * P[l] - l * P[l - 1]) / (l + 1);
        dP[l + 1] = dP[l - 1] + (2 * l + 1) * P[l];
    }
}

typedef struct {
    const orc_model *m;
    const double *cR, *cA, *scaler, *nn, *b1;
    int nR, nA, D, H, per_type;
} orc_params;

static void split_params(const orc_model *m, const double *p, orc_params *P)
{
    int T = m->n_types;
    P->m = m;
    P->nR = m->n_max_r + 1;
    P->nA = m->n_max_a + 1;
    P->D = P->nR + P->nA * m->l_max + (m->l_max_4b == 2 ? P->nA : 0) + (m->l_max_5b == 1 ? P->nA : 0);
    P->H = m->n_neurons;
    P->cR = p;
    P->cA = P->cR + (size_t)T * T * P->nR * (m->basis_r + 1);
    P->scaler = P->cA + (size_t)T * T * P->nA * (m->basis_a + 1);
    P->nn = P->scaler + P->D;
    P->per_type = P->H * P->D + 3 * P->H;
    P->b1 = P->nn + (size_t)T * P->per_type;
}

#define ORC_MAXB 32   /* max basis functions / radial functions / l */

/* D^i: radial D_n = sum_j g^R_n(r_ij); angular D_nl = sum_j sum_k g^A_n(r_ij) g^A_n(r_ik) P_l(cos th_jk),
 * l = 1..l_max, j = k terms included; order: radial first, then nu = nR + n*l_max + (l-1). */
static void descriptor_of_atom(const orc_params *P, const int32_t *types, const orc_nlist *nl, int64_t i, double *D)
{
    const orc_model *m = P->m;
    int ti = types[i];
    for (int v = 0; v < P->D; ++v) D[v] = 0.0;
    int64_t b = nl->start[i], e = nl->start[i + 1];
    double f[ORC_MAXB], df[ORC_MAXB], g[ORC_MAXB], dg[ORC_MAXB];
    /* radial */
    for (int64_t p = b; p < e; ++p) {
        double r = nl->d[4 * p + 3];
        radial_basis(r, m->rc_r, m->basis_r, f, df);
        g_functions(P->cR, m->n_types, ti, types[nl->j[p]], P->nR, m->basis_r, f, df, g, dg);
        for (int n = 0; n < P->nR; ++n) D[n] += g[n];
    }
    /* angular: gather the neighbours inside rc_a */
    int64_t na = 0;
    for (int64_t p = b; p < e; ++p) if (nl->d[4 * p + 3] < m->rc_a) ++na;
    if (na == 0) return;
    double *ga = (double *)malloc(sizeof(double) * na * P->nA);
    double *u = (double *)malloc(sizeof(double) * na * 3);
    int64_t q = 0;
    for (int64_t p = b; p < e; ++p) {
        double r = nl->d[4 * p + 3];
        if (r >= m->rc_a) continue;
        radial_basis(r, m->rc_a, m->basis_a, f, df);
        g_functions(P->cA, m->n_types, ti, types[nl->j[p]], P->nA, m->basis_a, f, df, g, dg);
        for (int n = 0; n < P->nA; ++n) ga[q * P->nA + n] = g[n];
        for (int a = 0; a < 3; ++a) u[3 * q + a] = nl->d[4 * p + a] / r;
        ++q;
    }
    double Pl[ORC_MAXB], dPl[ORC_MAXB];
    for (int64_t j = 0; j < na; ++j)
        for (int64_t k = 0; k < na; ++k) {
            double c = u[3 * j] * u[3 * k] + u[3 * j + 1] * u[3 * k + 1] + u[3 * j + 2] * u[3 * k + 2];
            legendre(c, m->l_max, Pl, dPl);
            for (int n = 0; n < P->nA; ++n)
                for (int l = 1; l <= m->l_max; ++l)
                    D[P->nR + n * m->l_max + (l - 1)] += ga[j * P->nA + n] * ga[k * P->nA + n] * Pl[l];
        }
    /* Higher-body terms of NEP4 (reading Z2), per radial channel n, appended after the 3-body block:
     *   4-body: q_n = tr(T_n^3),  T_n = sum_j g_n(r_ij) (rhat_ij rhat_ij^T - 1/3)   (the cubic invariant of the l = 2 moments;
     *           as a sum over neighbour triples: g_j g_k g_l [c_jk c_kl c_lj - (c_jk^2 + c_kl^2 + c_lj^2)/3 + 2/9])
     *   5-body: q_n = (w_n . w_n)^2,  w_n = sum_j g_n(r_ij) rhat_ij                (the l = 1 invariant squared;
     *           as a sum over neighbour quadruples: g_j g_k g_l g_m c_jk c_lm)                                        */
    int o4 = P->nR + P->nA * m->l_max, o5 = o4 + (m->l_max_4b == 2 ? P->nA : 0);
    for (int n = 0; n < P->nA; ++n) {
        double T[3][3] = {{0}}, w[3] = {0, 0, 0};
        for (int64_t j = 0; j < na; ++j) {
            double gj = ga[j * P->nA + n];
            for (int a = 0; a < 3; ++a) {
                w[a] += gj * u[3 * j + a];
                for (int c = 0; c < 3; ++c) T[a][c] += gj * (u[3 * j + a] * u[3 * j + c] - (a == c ? 1.0 / 3.0 : 0.0));
            }
        }
        if (m->l_max_4b == 2) {
            double t3 = 0.0;
            for (int a = 0; a < 3; ++a)
                for (int c = 0; c < 3; ++c)
                    for (int d = 0; d < 3; ++d) t3 += T[a][c] * T[c][d] * T[d][a];
            D[o4 + n] = t3;
        }
        if (m->l_max_5b == 1) {
            double w2 = w[0] * w[0] + w[1] * w[1] + w[2] * w[2];
            D[o5 + n] = w2 * w2;
        }
    }
    free(ga);
    free(u);
}

/* partial forces F_ij = sum_nu Fp_nu dD_nu/dr_ij for every neighbour (b..e) of atom i (Eq. 14, 17; S2):
 *   radial : dD_n/dr_ij  = g_n'(r_ij) rhat_ij
 *   angular: dD_nl/dr_ij = 2 sum_k g_n(r_ik) [ g_n'(r_ij) P_l(c_jk) rhat_ij
 *                                            + g_n(r_ij) P_l'(c_jk) (rhat_ik - c_jk rhat_ij) / r_ij ]
 * out: Fij[(p-b)*3 + a] */
static void partial_forces_of_atom(const orc_params *P, const int32_t *types, const orc_nlist *nl, int64_t i,
                                   const double *Fp, double *Fij)
{
    const orc_model *m = P->m;
    int ti = types[i];
    int64_t b = nl->start[i], e = nl->start[i + 1];
    double f[ORC_MAXB], df[ORC_MAXB], g[ORC_MAXB], dg[ORC_MAXB];
    for (int64_t p = b; p < e; ++p) {
        double r = nl->d[4 * p + 3];
        radial_basis(r, m->rc_r, m->basis_r, f, df);
        g_functions(P->cR, m->n_types, ti, types[nl->j[p]], P->nR, m->basis_r, f, df, g, dg);
        double s = 0.0;
        for (int n = 0; n < P->nR; ++n) s += Fp[n] * dg[n];
        for (int a = 0; a < 3; ++a) Fij[(p - b) * 3 + a] = s * nl->d[4 * p + a] / r;
    }
    int64_t na = 0;
    for (int64_t p = b; p < e; ++p) if (nl->d[4 * p + 3] < m->rc_a) ++na;
    if (na == 0) return;
    double *ga = (double *)malloc(sizeof(double) * na * P->nA);
    double *dga = (double *)malloc(sizeof(double) * na * P->nA);
    double *u = (double *)malloc(sizeof(double) * na * 3);
    double *ra = (double *)malloc(sizeof(double) * na);
    int64_t *idx = (int64_t *)malloc(sizeof(int64_t) * na);
    int64_t q = 0;
    for (int64_t p = b; p < e; ++p) {
        double r = nl->d[4 * p + 3];
        if (r >= m->rc_a) continue;
        radial_basis(r, m->rc_a, m->basis_a, f, df);
        g_functions(P->cA, m->n_types, ti, types[nl->j[p]], P->nA, m->basis_a, f, df, g, dg);
        for (int n = 0; n < P->nA; ++n) { ga[q * P->nA + n] = g[n]; dga[q * P->nA + n] = dg[n]; }
        for (int a = 0; a < 3; ++a) u[3 * q + a] = nl->d[4 * p + a] / r;
        ra[q] = r;
        idx[q] = p - b;
        ++q;
    }
    double Pl[ORC_MAXB], dPl[ORC_MAXB];
    for (int64_t j = 0; j < na; ++j) {
        double F[3] = {0, 0, 0};
        for (int64_t k = 0; k < na; ++k) {
            double c = u[3 * j] * u[3 * k] + u[3 * j + 1] * u[3 * k + 1] + u[3 * j + 2] * u[3 * k + 2];
            legendre(c, m->l_max, Pl, dPl);
            for (int n = 0; n < P->nA; ++n)
                for (int l = 1; l <= m->l_max; ++l) {
                    double fp = Fp[P->nR + n * m->l_max + (l - 1)];
                    double gk = ga[k * P->nA + n];
                    double t1 = 2.0 * fp * gk * dga[j * P->nA + n] * Pl[l];
                    double t2 = 2.0 * fp * gk * ga[j * P->nA + n] * dPl[l] / ra[j];
                    for (int a = 0; a < 3; ++a)
                        F[a] += t1 * u[3 * j + a] + t2 * (u[3 * k + a] - c * u[3 * j + a]);
                }
        }
        for (int a = 0; a < 3; ++a) Fij[idx[j] * 3 + a] += F[a];
    }
    /* higher-body terms (reading Z2): with S = T^2,
     *   d tr(T^3)/dr_ij = 3 [ g' rhat (rhat.S.rhat - tr S / 3) + (g / r) 2 (S rhat - rhat (rhat.S.rhat)) ]
     *   d (w.w)^2/dr_ij = 4 (w.w) [ g' rhat (w.rhat) + (g / r) (w - rhat (w.rhat)) ]                        */
    int o4 = P->nR + P->nA * m->l_max, o5 = o4 + (m->l_max_4b == 2 ? P->nA : 0);
    for (int n = 0; n < P->nA && (m->l_max_4b == 2 || m->l_max_5b == 1); ++n) {
        double T[3][3] = {{0}}, w[3] = {0, 0, 0}, S[3][3] = {{0}};
        for (int64_t j = 0; j < na; ++j) {
            double gj = ga[j * P->nA + n];
            for (int a = 0; a < 3; ++a) {
                w[a] += gj * u[3 * j + a];
                for (int c = 0; c < 3; ++c) T[a][c] += gj * (u[3 * j + a] * u[3 * j + c] - (a == c ? 1.0 / 3.0 : 0.0));
            }
        }
        for (int a = 0; a < 3; ++a)
            for (int c = 0; c < 3; ++c)
                for (int d = 0; d < 3; ++d) S[a][c] += T[a][d] * T[d][c];
        double trS = S[0][0] + S[1][1] + S[2][2], w2 = w[0] * w[0] + w[1] * w[1] + w[2] * w[2];
        for (int64_t j = 0; j < na; ++j) {
            const double *uj = u + 3 * j;
            double gj = ga[j * P->nA + n], dgj = dga[j * P->nA + n];
            double Su[3], uSu = 0.0, wu = 0.0;
            for (int a = 0; a < 3; ++a) {
                Su[a] = S[a][0] * uj[0] + S[a][1] * uj[1] + S[a][2] * uj[2];
                wu += w[a] * uj[a];
            }
            for (int a = 0; a < 3; ++a) uSu += uj[a] * Su[a];
            for (int a = 0; a < 3; ++a) {
                double f = 0.0;
                if (m->l_max_4b == 2)
                    f += Fp[o4 + n] * 3.0 * (dgj * uj[a] * (uSu - trS / 3.0) + gj / ra[j] * 2.0 * (Su[a] - uj[a] * uSu));
                if (m->l_max_5b == 1)
                    f += Fp[o5 + n] * 4.0 * w2 * (dgj * uj[a] * wu + gj / ra[j] * (w[a] - uj[a] * wu));
                Fij[idx[j] * 3 + a] += f;
            }
        }
    }
    free(ga); free(dga); free(u); free(ra); free(idx);
}

/* NN (Eq. 1, :58-60; S4, S5): x = s.D; h = tanh(w0 x - b0); U = w1U.h - b1U; q = w1q.h - b1q.
 * Also dU/dD_nu and dq/dD_nu (scaler included). */
static void nn_of_atom(const orc_params *P, int ti, const double *D, double *U, double *q, double *dUdD, double *dqdD)
{
    int H = P->H, Dn = P->D;
    const double *w0 = P->nn + (size_t)ti * P->per_type;
    const double *b0 = w0 + (size_t)H * Dn;
    const double *w1U = b0 + H;
    const double *w1q = w1U + H;
    double u = 0.0, qq = 0.0;
    for (int v = 0; v < Dn; ++v) dUdD[v] = dqdD[v] = 0.0;
    for (int mu = 0; mu < H; ++mu) {
        double z = 0.0;
        for (int v = 0; v < Dn; ++v) z += w0[mu * Dn + v] * (P->scaler[v] * D[v]);
        z -= b0[mu];
        double h = tanh(z);
        u += w1U[mu] * h;
        qq += w1q[mu] * h;
        double dh = 1.0 - h * h;
        for (int v = 0; v < Dn; ++v) {
            dUdD[v] += w1U[mu] * dh * w0[mu * Dn + v] * P->scaler[v];
            dqdD[v] += w1q[mu] * dh * w0[mu * Dn + v] * P->scaler[v];
        }
    }
    *U = u - P->b1[0];
    *q = qq - P->b1[1];
}

/* exported: unscaled descriptors of all atoms, D[N][n_desc] */
int orc_descriptors(const orc_model *m, const double *params, int64_t n, const double *pos, const int32_t *types,
                    const double *box, int use_bins, double *D)
{
    orc_params P;
    split_params(m, params, &P);
    if (m->rc_a > m->rc_r || P.nR > ORC_MAXB || P.nA > ORC_MAXB || m->basis_r + 1 > ORC_MAXB ||
        m->basis_a + 1 > ORC_MAXB || m->l_max + 1 > ORC_MAXB) return -2;
    double *w = (double *)malloc(sizeof(double) * 3 * (n > 0 ? n : 1));
    wrap_positions(n, pos, box, w);
    orc_nlist nl;
    if (build_nlist(n, w, box, m->rc_r, use_bins, &nl)) { free(w); return -1; }
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < n; ++i) descriptor_of_atom(&P, types, &nl, i, D + i * P.D);
    nlist_free(&nl);
    free(w);
    return 0;
}

/* ------------------------------------------------------------------------- */
/* PPPM building blocks (S10, G2, S11)                                        */
/* ------------------------------------------------------------------------- */
/* centred cardinal B-spline of order 5: weights on mesh offsets -2..2 around the nearest
 * mesh point; dx = u - round(u) in [-1/2, 1/2)  (S10) */
void orc_bspline5(double dx, double *w)
{
    double d2 = dx * dx, d3 = d2 * dx, d4 = d2 * d2;
    w[0] = (1.0 - 8.0 * dx + 24.0 * d2 - 32.0 * d3 + 16.0 * d4) / 384.0;
    w[1] = (19.0 - 44.0 * dx + 24.0 * d2 + 16.0 * d3 - 16.0 * d4) / 96.0;
    w[2] = (115.0 - 120.0 * d2 + 48.0 * d4) / 192.0;
    w[3] = (19.0 + 44.0 * dx + 24.0 * d2 - 16.0 * d3 - 16.0 * d4) / 96.0;
    w[4] = (1.0 + 8.0 * dx + 24.0 * d2 + 32.0 * d3 + 16.0 * d4) / 384.0;
}

/* denominator polynomial of Eq. 36 (reading G2), z = sin(pi n / N) */
double orc_alias_denominator(double z)
{
    double z2 = z * z;
    return 1.0 - 5.0 / 3.0 * z2 + 7.0 / 9.0 * z2 * z2 - 17.0 / 189.0 * z2 * z2 * z2 + 2.0 / 2835.0 * z2 * z2 * z2 * z2;
}

/* in-place unnormalised complex FFT of length n (power of 2), stride in complex elements;
 * sign = -1: sum x e^{-2 pi i jk/n} (forward, S11); sign = +1: inverse, unnormalised */
static void fft1d(double *x, int n, int64_t stride, int sign)
{
    /* bit reversal */
    for (int i = 1, j = 0; i < n; ++i) {
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) {
            double tr = x[2 * i * stride], ti = x[2 * i * stride + 1];
            x[2 * i * stride] = x[2 * j * stride];
            x[2 * i * stride + 1] = x[2 * j * stride + 1];
            x[2 * j * stride] = tr;
            x[2 * j * stride + 1] = ti;
        }
    }
    for (int len = 2; len <= n; len <<= 1) {
        double ang = sign * 2.0 * ORC_PI / len;
        for (int i = 0; i < n; i += len)
            for (int k = 0; k < len / 2; ++k) {
                double wr = cos(ang * k), wi = sin(ang * k);
                double *a = x + 2 * (i + k) * stride, *b = x + 2 * (i + k + len / 2) * stride;
                double tr = b[0] * wr - b[1] * wi, ti = b[0] * wi + b[1] * wr;
                b[0] = a[0] - tr; b[1] = a[1] - ti;
                a[0] += tr; a[1] += ti;
            }
    }
}

/* 3-D transform of an interleaved complex array [n0][n1][n2] (last index fastest) */
int orc_fft3d(double *x, int n0, int n1, int n2, int sign)
{
    int dims[3] = {n0, n1, n2};
    for (int a = 0; a < 3; ++a)
        if (dims[a] < 1 || (dims[a] & (dims[a] - 1))) return -2;
#pragma omp parallel for schedule(static)
    for (int64_t l = 0; l < (int64_t)n0 * n1; ++l) fft1d(x + 2 * l * n2, n2, 1, sign);
#pragma omp parallel for schedule(static)
    for (int64_t l = 0; l < (int64_t)n0 * n2; ++l) {
        int64_t i0 = l / n2, i2 = l % n2;
        fft1d(x + 2 * (i0 * n1 * (int64_t)n2 + i2), n1, n2, sign);
    }
#pragma omp parallel for schedule(static)
    for (int64_t l = 0; l < (int64_t)n1 * n2; ++l) fft1d(x + 2 * l, n0, (int64_t)n1 * n2, sign);
    return 0;
}

static double sinc(double x) { return x == 0.0 ? 1.0 : sin(x) / x; }

/* ------------------------------------------------------------------------- */
/* electrostatics for given charges                                           */
/* ------------------------------------------------------------------------- */
/* U[0..2] = U^r, U^k, U^s;  phi[N] = dU^ES/dq_i;  F[3][N] static force;  W[9] static virial.
 * w = wrapped positions.  nl = radial neighbour list (rc = rc_r) or NULL when mode == 2. */
static int electrostatics(int64_t n, const double *w, const double *q, const double *box, double rc, int mode,
                          const orc_es *es, const orc_nlist *nl, double *U, double *phi, double *F, double *W,
                          double *rho_out, double *Wat)
{
    const double K = ORC_K_COULOMB;
    double alpha = es->alpha > 0.0 ? es->alpha : ORC_PI / rc;
    double vol = fabs(det3(box));
    U[0] = U[1] = U[2] = 0.0;
    for (int64_t i = 0; i < n; ++i) phi[i] = 0.0;
    for (int64_t i = 0; i < 3 * n; ++i) F[i] = 0.0;
    for (int a = 0; a < 9; ++a) W[a] = 0.0;
    if (Wat) for (int64_t i = 0; i < 9 * n; ++i) Wat[i] = 0.0;
    if (es->method == 0) return 0;

    if (mode == 1) {
        /* Eq. 6 (G1), bracket of Eq. 16, Eq. 15 through Eq. 11, Eq. 12 */
        double Ur = 0.0, Wr[9] = {0};
        for (int64_t i = 0; i < n; ++i) {
            for (int64_t p = nl->start[i]; p < nl->start[i + 1]; ++p) {
                const double *d = nl->d + 4 * p;
                double r = d[3];
                int64_t j = nl->j[p];
                double e = erfc(alpha * r) / r;
                Ur += 0.5 * K * q[i] * q[j] * e;
                phi[i] += K * q[j] * e;
                double br = (2.0 * alpha / sqrt(ORC_PI) * r * exp(-alpha * alpha * r * r) + erfc(alpha * r)) / (r * r * r);
                for (int a = 0; a < 3; ++a) {
                    F[a * n + i] += -K * q[i] * q[j] * br * d[a];
                    for (int c = 0; c < 3; ++c) {
                        Wr[3 * a + c] += 0.5 * K * q[i] * q[j] * br * d[a] * d[c];
                        /* Eq. 12 with Eq. 15: W_i = sum_j r_ij (x) F_ji^{r,static}, F_ji = +1/2 K q_i q_j [..] r_ij / r^3 */
                        if (Wat) Wat[(3 * a + c) * n + i] += 0.5 * K * q[i] * q[j] * br * d[a] * d[c];
                    }
                }
            }
        }
        U[0] = Ur;
        for (int a = 0; a < 9; ++a) W[a] += Wr[a];
        /* Eq. 10, Eq. 23 */
        for (int64_t i = 0; i < n; ++i) {
            U[2] += -K * alpha / sqrt(ORC_PI) * q[i] * q[i];
            phi[i] += -2.0 * K * alpha / sqrt(ORC_PI) * q[i];
        }
    }

    if (es->method == 1) {
        /* Ewald reciprocal part: Eq. 7-9, 18, 19, 21-22; full sphere of k != 0 */
        double inv[9];
        inv3(box, inv); /* k = 2 pi (n0 inv[:,0] + n1 inv[:,1] + n2 inv[:,2]) */
        double kmax = 2.0 * ORC_PI * alpha;
        int nmax[3];
        for (int a = 0; a < 3; ++a) {
            if (es->ewald_nmax2 > 0) nmax[a] = (int)floor(sqrt((double)es->ewald_nmax2));
            else {
                double len = sqrt(box[3 * a] * box[3 * a] + box[3 * a + 1] * box[3 * a + 1] + box[3 * a + 2] * box[3 * a + 2]);
                nmax[a] = (int)ceil(kmax * len / (2.0 * ORC_PI)) + 1;
            }
        }
        int64_t nk_box = (int64_t)(2 * nmax[0] + 1) * (2 * nmax[1] + 1) * (2 * nmax[2] + 1);
        double Uk = 0.0, Wk[9] = {0};
#pragma omp parallel
        {
            double *phi_l = (double *)calloc(n > 0 ? n : 1, sizeof(double));
            double *F_l = (double *)calloc(n > 0 ? 3 * n : 1, sizeof(double));
            double *Wat_l = Wat ? (double *)calloc(n > 0 ? 9 * n : 1, sizeof(double)) : 0;
            double Uk_l = 0.0, Wk_l[9] = {0};
#pragma omp for schedule(dynamic, 8)
            for (int64_t t = 0; t < nk_box; ++t) {
                int n0 = (int)(t / ((2 * nmax[1] + 1) * (2 * nmax[2] + 1))) - nmax[0];
                int n1 = (int)((t / (2 * nmax[2] + 1)) % (2 * nmax[1] + 1)) - nmax[1];
                int n2 = (int)(t % (2 * nmax[2] + 1)) - nmax[2];
                if (n0 == 0 && n1 == 0 && n2 == 0) continue;
                double k[3];
                for (int a = 0; a < 3; ++a)
                    k[a] = 2.0 * ORC_PI * (n0 * inv[3 * a + 0] + n1 * inv[3 * a + 1] + n2 * inv[3 * a + 2]);
                double k2 = k[0] * k[0] + k[1] * k[1] + k[2] * k[2];
                if (es->ewald_nmax2 > 0) { if (n0 * n0 + n1 * n1 + n2 * n2 > es->ewald_nmax2) continue; }
                else if (k2 > kmax * kmax * (1.0 + 1e-12)) continue;
                double G = 2.0 * ORC_PI / vol * exp(-k2 / (4.0 * alpha * alpha)) / k2;   /* Eq. 9 */
                double Sr = 0.0, Si = 0.0;                                             /* Eq. 8 */
                for (int64_t i = 0; i < n; ++i) {
                    double ph = k[0] * w[i] + k[1] * w[n + i] + k[2] * w[2 * n + i];
                    Sr += q[i] * cos(ph);
                    Si -= q[i] * sin(ph);
                }
                double S2 = Sr * Sr + Si * Si;
                Uk_l += K * G * S2;                                                     /* Eq. 7 */
                double bfac = 2.0 / (4.0 * alpha * alpha) + 2.0 / k2;                   /* Eq. 21 */
                for (int a = 0; a < 3; ++a)
                    for (int c = 0; c < 3; ++c)
                        Wk_l[3 * a + c] += K * G * S2 * ((a == c ? 1.0 : 0.0) - bfac * k[a] * k[c]); /* Eq. 22 */
                for (int64_t i = 0; i < n; ++i) {
                    double ph = k[0] * w[i] + k[1] * w[n + i] + k[2] * w[2 * n + i];
                    double c = cos(ph), s = sin(ph);
                    double re = Sr * c - Si * s;  /* Re[S e^{ik.r}] */
                    double im = Sr * s + Si * c;  /* Im[S e^{ik.r}] */
                    phi_l[i] += 2.0 * K * G * re;                                       /* bracket of Eq. 19 */
                    for (int a = 0; a < 3; ++a) F_l[a * n + i] += 2.0 * K * q[i] * G * k[a] * im; /* Eq. 18 */
                    if (Wat_l)                                                          /* Eq. 20, real part (reading G4) */
                        for (int a = 0; a < 3; ++a)
                            for (int cc = 0; cc < 3; ++cc)
                                Wat_l[(3 * a + cc) * n + i] += K * G * q[i] * re * ((a == cc ? 1.0 : 0.0) - bfac * k[a] * k[cc]);
                }
            }
#pragma omp critical
            {
                Uk += Uk_l;
                for (int a = 0; a < 9; ++a) Wk[a] += Wk_l[a];
                for (int64_t i = 0; i < n; ++i) phi[i] += phi_l[i];
                for (int64_t i = 0; i < 3 * n; ++i) F[i] += F_l[i];
                if (Wat_l) for (int64_t i = 0; i < 9 * n; ++i) Wat[i] += Wat_l[i];
            }
            free(phi_l);
            free(F_l);
            free(Wat_l);
        }
        U[1] = Uk;
        for (int a = 0; a < 9; ++a) W[a] += Wk[a];
    } else if (es->method == 2) {
        /* PPPM: Eq. 34-38, order 5, any cell (:104 "k from the reciprocal basis vectors"): the mesh lives in fractional
         * coordinates, mesh point s = (s_0 a + s_1 b + s_2 c) / N, and k = 2 pi (n_0 b*_0 + n_1 b*_1 + n_2 b*_2) */
        if (es->order != 5) return -3;
        int N[3] = {es->grid[0], es->grid[1], es->grid[2]};
        double inv[9];
        inv3(box, inv);          /* fractional coordinate f_b = sum_a r_a inv[3 a + b];  k_a = 2 pi sum_b n_b inv[3 a + b] */
        int64_t ng = (int64_t)N[0] * N[1] * N[2];
        double *rho = (double *)calloc(2 * ng, sizeof(double));   /* complex */
        double *fld = (double *)malloc(sizeof(double) * 2 * ng);
        double *mesh[4];                                          /* Phi, Ex, Ey, Ez (real) */
        for (int c = 0; c < 4; ++c) mesh[c] = (double *)malloc(sizeof(double) * ng);
        if (!rho || !fld || !mesh[3]) return -1;
        /* charge assignment, Eq. 35 (S10): mesh point r_s = (s_x h_x, s_y h_y, s_z h_z) */
        for (int64_t i = 0; i < n; ++i) {
            int i0[3];
            double wt[3][5];
            for (int a = 0; a < 3; ++a) {
                double u = (w[i] * inv[a] + w[n + i] * inv[3 + a] + w[2 * n + i] * inv[6 + a]) * N[a];
                i0[a] = (int)floor(u + 0.5);
                orc_bspline5(u - i0[a], wt[a]);
            }
            for (int a = 0; a < 5; ++a)
                for (int b = 0; b < 5; ++b)
                    for (int c = 0; c < 5; ++c) {
                        int64_t s0 = ((i0[0] + a - 2) % N[0] + N[0]) % N[0];
                        int64_t s1 = ((i0[1] + b - 2) % N[1] + N[1]) % N[1];
                        int64_t s2 = ((i0[2] + c - 2) % N[2] + N[2]) % N[2];
                        rho[2 * ((s0 * N[1] + s1) * N[2] + s2)] += q[i] * wt[0][a] * wt[1][b] * wt[2][c];
                    }
        }
        if (rho_out) for (int64_t s = 0; s < ng; ++s) rho_out[s] = rho[2 * s];
        /* S(k) on the mesh: forward FFT (:302, S11) */
        orc_fft3d(rho, N[0], N[1], N[2], -1);
        /* Eq. 34, 36 (G2), 22 with G^opt */
        double Uk = 0.0, Wk[9] = {0};
        double *Gopt = (double *)malloc(sizeof(double) * ng);
        for (int64_t m0 = 0; m0 < N[0]; ++m0)
            for (int64_t m1 = 0; m1 < N[1]; ++m1)
                for (int64_t m2 = 0; m2 < N[2]; ++m2) {
                    int64_t s = (m0 * N[1] + m1) * N[2] + m2;
                    int64_t mm[3] = {m0, m1, m2};
                    double k[3] = {0.0, 0.0, 0.0}, num = 1.0, den = 1.0;
                    for (int b = 0; b < 3; ++b) {
                        int64_t nb = mm[b] < N[b] / 2 ? mm[b] : mm[b] - N[b];   /* -N/2 <= n < N/2 (:285) */
                        for (int a = 0; a < 3; ++a) k[a] += 2.0 * ORC_PI * nb * inv[3 * a + b];
                        double x = ORC_PI * nb / N[b];
                        num *= pow(sinc(x), 5);
                        den *= orc_alias_denominator(sin(x));
                    }
                    double k2 = k[0] * k[0] + k[1] * k[1] + k[2] * k[2];
                    if (k2 == 0.0) { Gopt[s] = 0.0; continue; }
                    double G = 2.0 * ORC_PI / vol * exp(-k2 / (4.0 * alpha * alpha)) / k2;
                    Gopt[s] = G * num * num / (den * den);
                    double S2 = rho[2 * s] * rho[2 * s] + rho[2 * s + 1] * rho[2 * s + 1];
                    Uk += K * Gopt[s] * S2;
                    double bfac = 2.0 / (4.0 * alpha * alpha) + 2.0 / k2;
                    for (int a = 0; a < 3; ++a)
                        for (int c = 0; c < 3; ++c)
                            Wk[3 * a + c] += K * Gopt[s] * S2 * ((a == c ? 1.0 : 0.0) - bfac * k[a] * k[c]);
                }
        U[1] = Uk;
        for (int a = 0; a < 9; ++a) W[a] += Wk[a];
        /* F^-1[S G^opt] (Eq. 38) and F^-1[i k_a S G^opt] (Eq. 37): four inverse FFTs (:302) */
        for (int comp = 0; comp < 4; ++comp) {
            for (int64_t m0 = 0; m0 < N[0]; ++m0)
                for (int64_t m1 = 0; m1 < N[1]; ++m1)
                    for (int64_t m2 = 0; m2 < N[2]; ++m2) {
                        int64_t s = (m0 * N[1] + m1) * N[2] + m2;
                        double re = rho[2 * s] * Gopt[s], im = rho[2 * s + 1] * Gopt[s];
                        if (comp == 0) { fld[2 * s] = re; fld[2 * s + 1] = im; }
                        else {
                            int a = comp - 1;
                            int64_t mm[3] = {m0, m1, m2};
                            double ka = 0.0;
                            for (int b = 0; b < 3; ++b) {
                                int64_t nb = mm[b] < N[b] / 2 ? mm[b] : mm[b] - N[b];
                                if (2 * nb == -(int64_t)N[b]) nb = 0;          /* S11: the Nyquist index carries no gradient */
                                ka += 2.0 * ORC_PI * nb * inv[3 * a + b];
                            }
                            fld[2 * s] = -ka * im;      /* i k (re + i im) */
                            fld[2 * s + 1] = ka * re;
                        }
                    }
            orc_fft3d(fld, N[0], N[1], N[2], +1);
            for (int64_t s = 0; s < ng; ++s) mesh[comp][s] = fld[2 * s];
        }
        /* back-interpolation with the same W */
        for (int64_t i = 0; i < n; ++i) {
            int i0[3];
            double wt[3][5];
            for (int a = 0; a < 3; ++a) {
                double u = (w[i] * inv[a] + w[n + i] * inv[3 + a] + w[2 * n + i] * inv[6 + a]) * N[a];
                i0[a] = (int)floor(u + 0.5);
                orc_bspline5(u - i0[a], wt[a]);
            }
            double acc[4] = {0, 0, 0, 0};
            for (int a = 0; a < 5; ++a)
                for (int b = 0; b < 5; ++b)
                    for (int c = 0; c < 5; ++c) {
                        int64_t s0 = ((i0[0] + a - 2) % N[0] + N[0]) % N[0];
                        int64_t s1 = ((i0[1] + b - 2) % N[1] + N[1]) % N[1];
                        int64_t s2 = ((i0[2] + c - 2) % N[2] + N[2]) % N[2];
                        double ww = wt[0][a] * wt[1][b] * wt[2][c];
                        for (int comp = 0; comp < 4; ++comp) acc[comp] += ww * mesh[comp][(s0 * N[1] + s1) * N[2] + s2];
                    }
            phi[i] += 2.0 * K * acc[0];                                       /* bracket of Eq. 38 */
            for (int a = 0; a < 3; ++a) F[a * n + i] += -2.0 * K * q[i] * acc[1 + a]; /* Eq. 37 */
        }
        if (Wat) {
            /* Eq. 39: W_i^{k,static} = K q_i sum_s W(r_i - r_s) F^-1[S G^opt B]_s -- six inverse FFTs (:302), one per
             * independent component of B (Eq. 21; true k in B, all mesh k != 0 as in Eq. 34) */
            static const int comp_ab[6][2] = {{0, 0}, {1, 1}, {2, 2}, {0, 1}, {0, 2}, {1, 2}};
            for (int comp = 0; comp < 6; ++comp) {
                int a = comp_ab[comp][0], b = comp_ab[comp][1];
                for (int64_t m0 = 0; m0 < N[0]; ++m0)
                    for (int64_t m1 = 0; m1 < N[1]; ++m1)
                        for (int64_t m2 = 0; m2 < N[2]; ++m2) {
                            int64_t s = (m0 * N[1] + m1) * N[2] + m2;
                            int64_t mm[3] = {m0, m1, m2};
                            double k[3] = {0.0, 0.0, 0.0};
                            for (int c = 0; c < 3; ++c) {
                                int64_t nc = mm[c] < N[c] / 2 ? mm[c] : mm[c] - N[c];
                                for (int d = 0; d < 3; ++d) k[d] += 2.0 * ORC_PI * nc * inv[3 * d + c];
                            }
                            double k2 = k[0] * k[0] + k[1] * k[1] + k[2] * k[2];
                            double Bab = 0.0;
                            if (k2 > 0.0) Bab = (a == b ? 1.0 : 0.0) - (2.0 / (4.0 * alpha * alpha) + 2.0 / k2) * k[a] * k[b];
                            fld[2 * s] = rho[2 * s] * Gopt[s] * Bab;
                            fld[2 * s + 1] = rho[2 * s + 1] * Gopt[s] * Bab;
                        }
                orc_fft3d(fld, N[0], N[1], N[2], +1);
                for (int64_t i = 0; i < n; ++i) {
                    int i0[3];
                    double wt[3][5];
                    for (int c = 0; c < 3; ++c) {
                        double u = (w[i] * inv[c] + w[n + i] * inv[3 + c] + w[2 * n + i] * inv[6 + c]) * N[c];
                        i0[c] = (int)floor(u + 0.5);
                        orc_bspline5(u - i0[c], wt[c]);
                    }
                    double acc = 0.0;
                    for (int aa = 0; aa < 5; ++aa)
                        for (int bb = 0; bb < 5; ++bb)
                            for (int cc = 0; cc < 5; ++cc) {
                                int64_t s0 = ((i0[0] + aa - 2) % N[0] + N[0]) % N[0];
                                int64_t s1 = ((i0[1] + bb - 2) % N[1] + N[1]) % N[1];
                                int64_t s2 = ((i0[2] + cc - 2) % N[2] + N[2]) % N[2];
                                acc += wt[0][aa] * wt[1][bb] * wt[2][cc] * fld[2 * ((s0 * N[1] + s1) * N[2] + s2)];
                            }
                    Wat[(3 * a + b) * n + i] += K * q[i] * acc;
                    if (a != b) Wat[(3 * b + a) * n + i] += K * q[i] * acc;
                }
            }
        }
        free(rho); free(fld); free(Gopt);
        for (int c = 0; c < 4; ++c) free(mesh[c]);
    } else {
        return -3;
    }
    return 0;
}

/* exported: electrostatics of FIXED charges (the static-charge pins: Madelung, brute-force image sum...) */
int orc_electrostatics(int64_t n, const double *pos, const double *q, const double *box, double rc, int mode,
                       const orc_es *es, double *U3, double *phi, double *F, double *W, double *rho, double *Wat)
{
    double *w = (double *)malloc(sizeof(double) * 3 * (n > 0 ? n : 1));
    wrap_positions(n, pos, box, w);
    orc_nlist nl;
    memset(&nl, 0, sizeof(nl));
    if (mode == 1 && build_nlist(n, w, box, rc, 1, &nl)) { free(w); return -1; }
    int rcode = electrostatics(n, w, q, box, rc, mode, es, mode == 1 ? &nl : 0, U3, phi, F, W, rho, Wat);
    if (mode == 1) nlist_free(&nl);
    free(w);
    return rcode;
}

/* ------------------------------------------------------------------------- */
/* the whole force evaluation                        */
/* ------------------------------------------------------------------------- */
/* energy[5] = {U^tot, U^NEP, U^r, U^k, U^s};  forces[3][N];  virial[9];  charges[N];  bec[9][N] or NULL;
 * virial_atom[9][N] or NULL: per-atom virial, W_i = sum_j r_ij (x) F_ji (Eq. 12) + W_i^{k,static} (Eq. 20 / Eq. 39) */
int orc_compute(const orc_model *m, const double *params, const orc_es *es, int64_t n, const double *pos,
                const int32_t *types, const double *box, int use_bins, double *energy, double *forces,
                double *virial, double *charges, double *bec, const orc_debug *dbg, double *virial_atom)
{
    orc_params P;
    split_params(m, params, &P);
    if (m->rc_a > m->rc_r || P.nR > ORC_MAXB || P.nA > ORC_MAXB || m->basis_r + 1 > ORC_MAXB ||
        m->basis_a + 1 > ORC_MAXB || m->l_max + 1 > ORC_MAXB) return -2;
    if (n <= 0) return -2;
    int Dn = P.D;
    /* 1. wrap, neighbours */
    double *w = (double *)malloc(sizeof(double) * 3 * n);
    wrap_positions(n, pos, box, w);
    orc_nlist nl;
    if (build_nlist(n, w, box, m->rc_r, use_bins, &nl)) { free(w); return -1; }
    /* 2.-3. descriptors, NN */
    double *D = (double *)malloc(sizeof(double) * n * Dn);
    double *dU = (double *)malloc(sizeof(double) * n * Dn);
    double *dq = (double *)malloc(sizeof(double) * n * Dn);
    double *Ui = (double *)malloc(sizeof(double) * n);
    double *q = (double *)malloc(sizeof(double) * n);
    double *phi = (double *)malloc(sizeof(double) * n);
    double *Fes = (double *)malloc(sizeof(double) * 3 * n);
    if (!D || !dU || !dq || !Ui || !q || !phi || !Fes) return -1;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < n; ++i) {
        descriptor_of_atom(&P, types, &nl, i, D + i * Dn);
        nn_of_atom(&P, types[i], D + i * Dn, Ui + i, q + i, dU + i * Dn, dq + i * Dn);
    }
    if (dbg && dbg->D) memcpy(dbg->D, D, sizeof(double) * n * Dn);
    if (dbg && dbg->U_i) memcpy(dbg->U_i, Ui, sizeof(double) * n);
    if (dbg && dbg->q_raw) memcpy(dbg->q_raw, q, sizeof(double) * n);
    /* 4. Eq. 33 (G3): q_i -> q_i + (Q - sum_j q_j) / N */
    double qsum = 0.0;
    for (int64_t i = 0; i < n; ++i) qsum += q[i];
    for (int64_t i = 0; i < n; ++i) q[i] += (m->q_total - qsum) / (double)n;
    /* 5.-6. electrostatics with the unscaled neutralised charges */
    double U3[3], Wes[9];
    int rcode = electrostatics(n, w, q, box, m->rc_r, m->mode, es, &nl, U3, phi, Fes, Wes, dbg ? dbg->rho : 0, virial_atom);
    if (rcode) return rcode;
    if (dbg && dbg->phi) memcpy(dbg->phi, phi, sizeof(double) * n);
    if (dbg && dbg->F_es) memcpy(dbg->F_es, Fes, sizeof(double) * 3 * n);
    /* S6: chain rule through Eq. 33 */
    double phibar = 0.0;
    for (int64_t i = 0; i < n; ++i) phibar += phi[i];
    phibar /= (double)n;
    /* 7. Fp = dU_i/dD + phi_eff dq_i/dD  (Eq. 14 + Eq. 17 folded, :140) */
    double *Fp = dU;
    for (int64_t i = 0; i < n; ++i)
        for (int v = 0; v < Dn; ++v) Fp[i * Dn + v] = dU[i * Dn + v] + (phi[i] - phibar) * dq[i * Dn + v];
    if (dbg && dbg->Fp) memcpy(dbg->Fp, Fp, sizeof(double) * n * Dn);
    /* 8.-9. F_i = sum_j (F_ij - F_ji) + static terms (Eq. 11); W = sum_i sum_j r_ij (x) F_ji (Eq. 12) */
    for (int64_t i = 0; i < 3 * n; ++i) forces[i] = Fes[i];
    double Wt[9];
    double Uzbl = 0.0;
    for (int a = 0; a < 9; ++a) Wt[a] = Wes[a];
    if (bec) for (int64_t i = 0; i < 9 * n; ++i) bec[i] = 0.0;
#pragma omp parallel
    {
        double Wl[9] = {0};
        double Uzl = 0.0;
#pragma omp for schedule(dynamic, 16)
        for (int64_t i = 0; i < n; ++i) {
            int64_t b = nl.start[i], cnt = nl.start[i + 1] - nl.start[i];
            double *Fij = (double *)malloc(sizeof(double) * 3 * (cnt > 0 ? cnt : 1));
            partial_forces_of_atom(&P, types, &nl, i, Fp + i * Dn, Fij);
            if (g_zbl.on) {
                /* ZBL site energy U_i = 1/2 sum_j U_ZBL(r_ij): partial force 1/2 U'(r_ij) rhat_ij (reading Z1) */
                for (int64_t p = 0; p < cnt; ++p) {
                    double r = nl.d[4 * (b + p) + 3], u, du;
                    if (r >= g_zbl.r2) continue;
                    orc_zbl_pair(r, g_zbl.Z[types[i]], g_zbl.Z[types[nl.j[b + p]]], g_zbl.r1, g_zbl.r2, &u, &du);
                    Uzl += 0.5 * u;
                    for (int a = 0; a < 3; ++a) Fij[3 * p + a] += 0.5 * du * nl.d[4 * (b + p) + a] / r;
                }
            }
            for (int64_t p = 0; p < cnt; ++p) {
                int64_t j = nl.j[b + p];
                for (int a = 0; a < 3; ++a) {
#pragma omp atomic
                    forces[a * n + i] += Fij[3 * p + a];      /* + F_ij on i           */
#pragma omp atomic
                    forces[a * n + j] -= Fij[3 * p + a];      /* - F_ij on j (= -F_ji term of atom j) */
                    /* this F_ij is the "F_ji" of atom j's sum in Eq. 12 with r_ji = -r_ij */
                    for (int c = 0; c < 3; ++c) {
                        Wl[3 * a + c] -= nl.d[4 * (b + p) + a] * Fij[3 * p + c];
                        if (virial_atom) {       /* W_j += r_ji (x) F_ij: the term belongs to atom j (Eq. 12) */
#pragma omp atomic
                            virial_atom[(3 * a + c) * n + j] -= nl.d[4 * (b + p) + a] * Fij[3 * p + c];
                        }
                    }
                }
            }
            if (bec) {
                /* 11. Eq. 28 (S12): partial c_ij = sqrt(eps_inf) dq_i/dr_ij contributes
                 * +1/2 r_ij (x) c_ij to Z_i and -1/2 r_ji (x) c_ij ... to Z_j, r_ji = -r_ij */
                double *cv = (double *)malloc(sizeof(double) * Dn);
                for (int v = 0; v < Dn; ++v) cv[v] = m->sqrt_eps_inf * dq[i * Dn + v];
                partial_forces_of_atom(&P, types, &nl, i, cv, Fij);
                for (int64_t p = 0; p < cnt; ++p) {
                    int64_t j = nl.j[b + p];
                    for (int a = 0; a < 3; ++a)
                        for (int c = 0; c < 3; ++c) {
                            double t = 0.5 * nl.d[4 * (b + p) + a] * Fij[3 * p + c];
#pragma omp atomic
                            bec[(3 * a + c) * n + i] += t;
#pragma omp atomic
                            bec[(3 * a + c) * n + j] -= t;
                        }
                }
                free(cv);
            }
            free(Fij);
        }
#pragma omp critical
        {
            for (int a = 0; a < 9; ++a) Wt[a] += Wl[a];
            Uzbl += Uzl;
        }
    }
    if (bec)
        for (int64_t i = 0; i < n; ++i)
            for (int a = 0; a < 3; ++a) bec[(3 * a + a) * n + i] += m->sqrt_eps_inf * q[i];   /* Eq. 24 */
    for (int a = 0; a < 9; ++a) virial[a] = Wt[a];
    /* 10. energies (Eq. 2, 3/5, 4) */
    double Unep = 0.0;
    for (int64_t i = 0; i < n; ++i) Unep += Ui[i];
    energy[1] = Unep;
    energy[2] = U3[0];
    energy[3] = U3[1];
    energy[4] = U3[2];
    energy[5] = Uzbl;
    energy[0] = Unep + U3[0] + U3[1] + U3[2] + Uzbl;
    for (int64_t i = 0; i < n; ++i) charges[i] = q[i];
    nlist_free(&nl);
    free(w); free(D); free(dU); free(dq); free(Ui); free(q); free(phi); free(Fes);
    return 0;
}

/* ------------------------------------------------------------------------- */
/* ZBL core repulsion (reading Z1; the paper defers to the NEP papers, :39)      */
/* ------------------------------------------------------------------------- */
/* U_ZBL(r) = K Z_i Z_j / r * phi(r / a) * f_sw(r),   a = 0.46850 / (Z_i^0.23 + Z_j^0.23) Angstrom,
 * phi(x) = 0.18175 e^{-3.19980 x} + 0.50986 e^{-0.94229 x} + 0.28022 e^{-0.40290 x} + 0.02817 e^{-0.20162 x}
 * (the universal screening function of Ziegler, Biersack and Littmark),
 * f_sw = 1 for r < r_1, 1/2 [1 + cos(pi (r - r_1) / (r_2 - r_1))] for r_1 <= r < r_2, 0 beyond.
 * The term enters as a site energy U_i^ZBL = 1/2 sum_j U_ZBL(r_ij), i.e. a partial force
 * dU_i/dr_ij = 1/2 U'_ZBL(r_ij) rhat_ij that goes through Eq. 11 and Eq. 12 like the NEP ones. */
void orc_zbl_pair(double r, double Zi, double Zj, double r1, double r2, double *u, double *du)
{
    static const double cphi[4] = {0.18175, 0.50986, 0.28022, 0.02817};
    static const double dphi[4] = {3.19980, 0.94229, 0.40290, 0.20162};
    *u = 0.0; *du = 0.0;
    if (r >= r2) return;
    double a = 0.46850 / (pow(Zi, 0.23) + pow(Zj, 0.23));
    double x = r / a, phi = 0.0, dphidr = 0.0;
    for (int k = 0; k < 4; ++k) {
        double e = cphi[k] * exp(-dphi[k] * x);
        phi += e;
        dphidr -= dphi[k] / a * e;
    }
    double fsw = 1.0, dfsw = 0.0;
    if (r >= r1) {
        double t = ORC_PI * (r - r1) / (r2 - r1);
        fsw = 0.5 * (1.0 + cos(t));
        dfsw = -0.5 * sin(t) * ORC_PI / (r2 - r1);
    }
    double c = ORC_K_COULOMB * Zi * Zj / r;              /* bare Coulomb repulsion of the nuclei */
    *u = c * phi * fsw;
    *du = -c / r * phi * fsw + c * dphidr * fsw + c * phi * dfsw;
}

/* ------------------------------------------------------------------------- */
/* Eq. 29-30 (PAPER.md :229-237): response to a homogeneous external field    */
/* ------------------------------------------------------------------------- */
/* bec[9][N] with entry (3 a + b) N + i = Z_{i,ab} (a: polarization component, b: displacement component, Eq. 27-28).
 * efield[3] or NULL -> fext[3][N];  vel[3][N] or NULL -> pdot[3]. */
void orc_response(int64_t n, const double *bec, const double *efield, const double *vel, double *fext, double *pdot)
{
    if (efield) {
        for (int64_t i = 0; i < n; ++i)
            for (int b = 0; b < 3; ++b) {
                double f = 0.0;
                for (int a = 0; a < 3; ++a) f += efield[a] * bec[(3 * a + b) * n + i];   /* Eq. 29 */
                fext[b * n + i] = f;
            }
    }
    if (vel) {
        for (int a = 0; a < 3; ++a) {
            double p = 0.0;
            for (int64_t i = 0; i < n; ++i)
                for (int b = 0; b < 3; ++b) p += bec[(3 * a + b) * n + i] * vel[b * n + i];   /* Eq. 30 */
            pdot[a] = p;
        }
    }
}
