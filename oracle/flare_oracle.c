/*
 * flare_oracle.c -- CPU ORACLE for the FLARE B2 force-field evaluation.
 *
 * THIS FILE IS TEST INFRASTRUCTURE.  It is a plain, slow, FP64, obviously-correct
 * restatement of what the hot path computes, written from the paper (arxiv 2204.12573,
 * cited below as P:L<line> of /root/reference/PAPER.md) and from SURVEY.md section 8(c)
 * (the READINGs R0..R16 where the paper is silent).  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code,
 * header, table or helper with the CUDA path under paper_2204_12573_b200/csrc/.
 *
 * What it computes, in the paper's order:
 *   1. local environment rho_i: all neighbours within r_cut            -> neighbours()
 *   2. ACE-B2 descriptor "constructed from an equivariant basis of spherical
 *      harmonics and radial functions"; radial = Chebyshev T_n times
 *      cosine cutoff (BASELINE.json north_star; R1,R2); real orthonormal Y_lm (R3)  -> env_A(), A_to_B()
 *   3. normalised descriptor d^ = d/||d||
 *   4. mapped mean  eps = d^T beta d^  (Eq. 1)   and
 *      mapped variance V = d^T gamma d^ (Eq. 2; gamma == north_star's Sigma)
 *   5. forces as minus the gradient of the predicted energy, "directly from grad d_i"
 *      -- the NAIVE route that P:L153 says FLARE avoids -- on purpose: the CUDA path
 *      uses the re-ordered summation, so the two derivations are independent.
 *   6. velocity-Verlet NVE step (north_star; R12,R13).
 *
 * Parity pins (tests/test_oracle_*.py, -m "not gpu"): descriptor dimension 420/112
 * (P:L155); T_n(cos t)=cos nt; f_c closed-form values; Y_lm vs scipy + orthonormality +
 * addition theorem; B2 vs the Legendre pair-sum closed form; E,V vs numpy x@M@x;
 * forces vs central finite differences of the total energy, beta=I => F=0, sum F = 0,
 * zero torque, perfect fcc => F=0; neighbours vs O(N^2) brute force and fcc 12+6 shells;
 * NVE drift ~ dt^2 and time reversal.  Nothing here is "parity unpinned".
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -fPIC -shared (no FMA contraction: R6).
 * Units (R13): Angstrom, eV, amu, fs.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_OK 0
#define ORACLE_ERR_ARG (-1)
#define ORACLE_ERR_BOX (-2)
#define ORACLE_ERR_OVERFLOW (-3)
#define ORACLE_ERR_NOMEM (-4)

#define LMAX_CAP 12

/* eV/amu expressed in Angstrom^2/fs^2 (R13): a = KAPPA * F / m */
static const double KAPPA = 9.648533212331e-3;

typedef struct {
    int S, n_max, l_max;
    const double *r_cut; /* [S*S] symmetric */
    const double *beta;  /* [S*P*P] row-major, one matrix per CENTRAL species (R10) */
    const double *sigma; /* [S*P*P] or NULL */
} model_t;

/* ------------------------------------------------------------------ sizes / indexing */

/* P = N_nu (N_nu+1)/2 * (l_max+1), N_nu = S*n_max.  Pinned by 420 and 112. */
int oracle_num_descriptors(int S, int n_max, int l_max)
{
    int Nv = S * n_max;
    return Nv * (Nv + 1) / 2 * (l_max + 1);
}

/* flat index of B[nu1<=nu2, l]: nu1 outer, nu2 middle, l inner (R4) */
int oracle_b2_index(int S, int n_max, int l_max, int v1, int v2, int l)
{
    int Nv = S * n_max, L = l_max + 1;
    return (v1 * Nv - v1 * (v1 - 1) / 2 + (v2 - v1)) * L + l;
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ------------------------------------------------------------------ radial basis (R1, R2) */

/* T_n(x), n = 0..n_max-1, and dT_n/dx = n U_{n-1}(x) */
void oracle_chebyshev(int n_max, double x, double *T, double *dT)
{
    double U[64];
    for (int n = 0; n < n_max; n++) {
        if (n == 0) { T[0] = 1.0; U[0] = 1.0; }
        else if (n == 1) { T[1] = x; U[1] = 2.0 * x; }
        else { T[n] = 2.0 * x * T[n - 1] - T[n - 2]; U[n] = 2.0 * x * U[n - 1] - U[n - 2]; }
    }
    for (int n = 0; n < n_max; n++) dT[n] = (n == 0) ? 0.0 : (double)n * U[n - 1];
}

/* cosine cutoff f_c(r) = 1/2 (1 + cos(pi r / r_c)) and its r-derivative */
double oracle_cutoff(double r, double rc, double *dfc)
{
    double a = M_PI * r / rc;
    if (dfc) *dfc = -(M_PI / (2.0 * rc)) * sin(a);
    return 0.5 * (1.0 + cos(a));
}

/* g~_n(r) = T_n(2r/r_c - 1) f_c(r) and d g~_n / dr */
void oracle_radial(int n_max, double r, double rc, double *g, double *dg)
{
    double T[64], dT[64], dfc;
    double x = 2.0 * r / rc - 1.0;
    double fc = oracle_cutoff(r, rc, &dfc);
    oracle_chebyshev(n_max, x, T, dT);
    for (int n = 0; n < n_max; n++) {
        g[n] = T[n] * fc;
        dg[n] = (2.0 / rc) * dT[n] * fc + T[n] * dfc;
    }
}

/* ------------------------------------------------------------------ real spherical harmonics (R3) */

static double factorial(int n)
{
    double f = 1.0;
    for (int i = 2; i <= n; i++) f *= (double)i;
    return f;
}

/*
 * Real orthonormal Y_lm at a UNIT vector u, index lm = l*l + (m + l), m = -l..l:
 *   Y_l0    =          K_l0 D_l^0(z)
 *   Y_l,+m  = sqrt(2)  K_lm D_l^m(z) Re[(x+iy)^m]
 *   Y_l,-m  = sqrt(2)  K_lm D_l^m(z) Im[(x+iy)^m]
 * K_lm = sqrt((2l+1)/(4 pi) (l-m)!/(l+m)!),  D_l^m = d^m P_l / dt^m (a polynomial), so
 * P_l^m(z) cos(m phi) = D_l^m(z) Re[(x+iy)^m] on the unit sphere and nothing divides by
 * sin(theta).  dY[lm*3+d] is the gradient of the POLYNOMIAL EXTENSION
 * Y~_lm(x,y,z) = K D_l^m(z) C_m(x,y) with respect to (x,y,z) at u; the caller projects it
 * onto the tangent plane.
 */
void oracle_ylm(int l_max, const double u[3], double *Y, double *dY)
{
    double D[LMAX_CAP + 1][LMAX_CAP + 3];
    double C[LMAX_CAP + 2], Sn[LMAX_CAP + 2];
    double x = u[0], y = u[1], z = u[2];
    /* D[l][m] = d^m P_l/dz^m by differentiating Bonnet's recurrence m times:
       l P_l = (2l-1) z P_{l-1} - (l-1) P_{l-2}
       => l D_l^m = (2l-1) (z D_{l-1}^m + m D_{l-1}^{m-1}) - (l-1) D_{l-2}^m            */
    for (int l = 0; l <= l_max; l++)
        for (int m = 0; m <= l_max + 2; m++) D[l][m] = 0.0;
    D[0][0] = 1.0;
    if (l_max >= 1) { D[1][0] = z; D[1][1] = 1.0; }
    for (int l = 2; l <= l_max; l++)
        for (int m = 0; m <= l; m++) {
            double lower = (m > 0) ? D[l - 1][m - 1] : 0.0;
            D[l][m] = ((2.0 * l - 1.0) * (z * D[l - 1][m] + m * lower) - (l - 1.0) * D[l - 2][m]) / (double)l;
        }
    /* C_m + i S_m = (x + i y)^m */
    C[0] = 1.0; Sn[0] = 0.0;
    for (int m = 1; m <= l_max; m++) {
        C[m] = x * C[m - 1] - y * Sn[m - 1];
        Sn[m] = x * Sn[m - 1] + y * C[m - 1];
    }
    for (int l = 0; l <= l_max; l++) {
        for (int m = 0; m <= l; m++) {
            double K = sqrt((2.0 * l + 1.0) / (4.0 * M_PI) * factorial(l - m) / factorial(l + m));
            double Dm = D[l][m], Dm1 = D[l][m + 1]; /* dD_l^m/dz = D_l^{m+1} */
            if (m == 0) {
                int i = l * l + l;
                Y[i] = K * Dm;
                if (dY) { dY[3 * i] = 0.0; dY[3 * i + 1] = 0.0; dY[3 * i + 2] = K * Dm1; }
            } else {
                double K2 = sqrt(2.0) * K;
                int ic = l * l + l + m, is = l * l + l - m;
                Y[ic] = K2 * Dm * C[m];
                Y[is] = K2 * Dm * Sn[m];
                if (dY) {
                    /* d(x+iy)^m/dx = m (x+iy)^{m-1};  d/dy = i m (x+iy)^{m-1} */
                    dY[3 * ic + 0] = K2 * Dm * m * C[m - 1];
                    dY[3 * ic + 1] = K2 * Dm * (-m * Sn[m - 1]);
                    dY[3 * ic + 2] = K2 * Dm1 * C[m];
                    dY[3 * is + 0] = K2 * Dm * m * Sn[m - 1];
                    dY[3 * is + 1] = K2 * Dm * m * C[m - 1];
                    dY[3 * is + 2] = K2 * Dm1 * Sn[m];
                }
            }
        }
    }
}

/* ------------------------------------------------------------------ geometry (R6, R7) */

static int box_is_orthorhombic(const double box[9])
{
    return box[1] == 0.0 && box[2] == 0.0 && box[3] == 0.0 && box[5] == 0.0 && box[6] == 0.0 && box[7] == 0.0 &&
           box[0] > 0.0 && box[4] > 0.0 && box[8] > 0.0;
}

/* canonical wrap into [0,L): x - L*floor(x/L); a result >= L (rounding) becomes 0 */
static double wrap1(double x, double L)
{
    double q = floor(x / L);
    double t = L * q;
    double w = x - t;
    if (w >= L) w = 0.0;
    if (w < 0.0) w = 0.0;
    return w;
}

void oracle_wrap(int64_t N, const double *pos, const double box[9], const int pbc[3], double *out)
{
    for (int64_t i = 0; i < N; i++)
        for (int d = 0; d < 3; d++)
            out[3 * i + d] = pbc[d] ? wrap1(pos[3 * i + d], box[4 * d]) : pos[3 * i + d];
}

/* canonical minimum-image displacement r_ij = x_j - x_i of WRAPPED positions */
static void min_image(const double *xi, const double *xj, const double box[9], const int pbc[3], double d[3])
{
    for (int k = 0; k < 3; k++) {
        double dx = xj[k] - xi[k];
        if (pbc[k]) {
            double L = box[4 * k], h = 0.5 * L;
            if (dx > h) dx = dx - L;
            else if (dx < -h) dx = dx + L;
        }
        d[k] = dx;
    }
}

/* d2 = ((dx*dx)+(dy*dy))+(dz*dz), each op rounded once (compiled with -ffp-contract=off) */
static double dist2(const double d[3])
{
    double a = d[0] * d[0], b = d[1] * d[1], c = d[2] * d[2];
    double s = a + b;
    return s + c;
}

static int check_system(const double box[9], const int pbc[3], int S, const double *r_cut)
{
    if (!box_is_orthorhombic(box)) return ORACLE_ERR_BOX;
    double rmax = 0.0;
    for (int a = 0; a < S; a++)
        for (int b = 0; b < S; b++) {
            if (r_cut[a * S + b] != r_cut[b * S + a] || !(r_cut[a * S + b] > 0.0)) return ORACLE_ERR_ARG;
            if (r_cut[a * S + b] > rmax) rmax = r_cut[a * S + b];
        }
    for (int d = 0; d < 3; d++)
        if (pbc[d] && box[4 * d] < 2.0 * rmax) return ORACLE_ERR_BOX; /* unique minimum image (R7) */
    return ORACLE_OK;
}

/* ------------------------------------------------------------------ neighbours (R5, R6) */

typedef struct {
    int64_t N;
    int64_t *off; /* [N+1] */
    int32_t *idx; /* [off[N]], each row sorted by j */
} nlist_t;

static void nlist_free(nlist_t *nl)
{
    free(nl->off); free(nl->idx);
    nl->off = NULL; nl->idx = NULL;
}

static int is_neighbour(int64_t i, int64_t j, const double *xw, const int32_t *types, const double box[9],
                        const int pbc[3], int S, const double *r_cut)
{
    double d[3];
    if (i == j) return 0;
    min_image(xw + 3 * i, xw + 3 * j, box, pbc, d);
    double rc = r_cut[types[i] * S + types[j]];
    return dist2(d) < rc * rc; /* strict (R6) */
}

static int cmp_i32(const void *a, const void *b)
{
    int32_t x = *(const int32_t *)a, y = *(const int32_t *)b;
    return (x > y) - (x < y);
}

/* method 0: brute force over all ordered pairs.  method 1: simple cell grid (checked
   against method 0 in the tests); candidates from a cell are tested with the SAME predicate. */
static int build_nlist(int64_t N, const double *xw, const int32_t *types, const double box[9], const int pbc[3],
                       int S, const double *r_cut, int method, nlist_t *nl)
{
    nl->N = N;
    nl->off = (int64_t *)calloc((size_t)N + 1, sizeof(int64_t));
    nl->idx = NULL;
    if (!nl->off) return ORACLE_ERR_NOMEM;

    int nc[3] = {1, 1, 1};
    double lo[3] = {0, 0, 0}, cw[3] = {1, 1, 1};
    int64_t *cell_start = NULL;
    int32_t *cell_atoms = NULL, *cell_of = NULL;
    if (method == 1) {
        double rmax = 0.0;
        for (int a = 0; a < S * S; a++) if (r_cut[a] > rmax) rmax = r_cut[a];
        for (int d = 0; d < 3; d++) {
            double len;
            if (pbc[d]) { lo[d] = 0.0; len = box[4 * d]; }
            else {
                double mn = 1e300, mx = -1e300;
                for (int64_t i = 0; i < N; i++) { double v = xw[3 * i + d]; if (v < mn) mn = v; if (v > mx) mx = v; }
                if (N == 0) { mn = 0; mx = 1; }
                lo[d] = mn; len = (mx - mn) + 1e-9 + 1e-12 * fabs(mx);
            }
            int n = (int)floor(len / rmax);
            if (n < 1) n = 1;
            if (n > 2048) n = 2048;
            nc[d] = n; cw[d] = len / n;
            if (pbc[d] && n < 3) method = 0; /* stencil would double count: fall back */
        }
    }
    if (method == 1) {
        int64_t ncell = (int64_t)nc[0] * nc[1] * nc[2];
        cell_start = (int64_t *)calloc((size_t)ncell + 1, sizeof(int64_t));
        cell_atoms = (int32_t *)malloc(sizeof(int32_t) * (size_t)(N > 0 ? N : 1));
        cell_of = (int32_t *)malloc(sizeof(int32_t) * (size_t)(N > 0 ? N : 1));
        if (!cell_start || !cell_atoms || !cell_of) return ORACLE_ERR_NOMEM;
        for (int64_t i = 0; i < N; i++) {
            int c[3];
            for (int d = 0; d < 3; d++) {
                int k = (int)floor((xw[3 * i + d] - lo[d]) / cw[d]);
                if (k < 0) k = 0;
                if (k >= nc[d]) k = nc[d] - 1;
                c[d] = k;
            }
            cell_of[i] = (int32_t)((c[2] * nc[1] + c[1]) * nc[0] + c[0]);
            cell_start[cell_of[i] + 1]++;
        }
        for (int64_t c = 0; c < ncell; c++) cell_start[c + 1] += cell_start[c];
        int64_t *fill = (int64_t *)malloc(sizeof(int64_t) * (size_t)(ncell > 0 ? ncell : 1));
        memcpy(fill, cell_start, sizeof(int64_t) * (size_t)ncell);
        for (int64_t i = 0; i < N; i++) cell_atoms[fill[cell_of[i]]++] = (int32_t)i;
        free(fill);
    }

    for (int pass = 0; pass < 2; pass++) {
        if (pass == 1) {
            for (int64_t i = 0; i < N; i++) nl->off[i + 1] += nl->off[i];
            nl->idx = (int32_t *)malloc(sizeof(int32_t) * (size_t)(nl->off[N] > 0 ? nl->off[N] : 1));
            if (!nl->idx) return ORACLE_ERR_NOMEM;
        }
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 64)
#endif
        for (int64_t i = 0; i < N; i++) {
            int64_t cnt = 0;
            int32_t *row = (pass == 1) ? nl->idx + nl->off[i] : NULL;
            if (method == 0) {
                for (int64_t j = 0; j < N; j++)
                    if (is_neighbour(i, j, xw, types, box, pbc, S, r_cut)) { if (row) row[cnt] = (int32_t)j; cnt++; }
            } else {
                int32_t ci = cell_of[i];
                int c0 = ci % nc[0], c1 = (ci / nc[0]) % nc[1], c2 = ci / (nc[0] * nc[1]);
                for (int a2 = -1; a2 <= 1; a2++)
                    for (int a1 = -1; a1 <= 1; a1++)
                        for (int a0 = -1; a0 <= 1; a0++) {
                            int k[3] = {c0 + a0, c1 + a1, c2 + a2};
                            int skip = 0;
                            for (int d = 0; d < 3; d++) {
                                if (pbc[d]) k[d] = (k[d] + nc[d]) % nc[d];
                                else if (k[d] < 0 || k[d] >= nc[d]) skip = 1;
                            }
                            if (skip) continue;
                            /* with nc<3 in a NON-periodic dim the same cell is never revisited
                               because out-of-range cells are skipped, but a0=-1 and a0=+1 could
                               still alias only under periodic wrap, which requires nc>=3 here */
                            int64_t c = ((int64_t)k[2] * nc[1] + k[1]) * nc[0] + k[0];
                            for (int64_t q = cell_start[c]; q < cell_start[c + 1]; q++) {
                                int64_t j = cell_atoms[q];
                                if (is_neighbour(i, j, xw, types, box, pbc, S, r_cut)) { if (row) row[cnt] = (int32_t)j; cnt++; }
                            }
                        }
                if (row) qsort(row, (size_t)cnt, sizeof(int32_t), cmp_i32);
            }
            if (pass == 0) nl->off[i + 1] = cnt;
        }
    }
    free(cell_start); free(cell_atoms); free(cell_of);
    return ORACLE_OK;
}

/* Exported: neighbour sets in the caller's atom order, row stride `cap`, rows sorted by j. */
int oracle_neighbors(int64_t N, const double *pos, const int32_t *types, const double box[9], const int pbc[3],
                     int S, const double *r_cut, int method, int32_t *cnt, int32_t *idx, int32_t cap)
{
    int rc = check_system(box, pbc, S, r_cut);
    if (rc) return rc;
    double *xw = (double *)malloc(sizeof(double) * 3 * (size_t)(N > 0 ? N : 1));
    if (!xw) return ORACLE_ERR_NOMEM;
    oracle_wrap(N, pos, box, pbc, xw);
    nlist_t nl;
    rc = build_nlist(N, xw, types, box, pbc, S, r_cut, method, &nl);
    if (rc == ORACLE_OK) {
        for (int64_t i = 0; i < N; i++) {
            int64_t m = nl.off[i + 1] - nl.off[i];
            cnt[i] = (int32_t)m;
            if (m > cap) { rc = ORACLE_ERR_OVERFLOW; continue; }
            for (int64_t q = 0; q < m; q++) idx[i * (int64_t)cap + q] = nl.idx[nl.off[i] + q];
        }
    }
    nlist_free(&nl);
    free(xw);
    return rc;
}

/* ------------------------------------------------------------------ descriptor (R3, R4) */

/* A[nu*L2 + lm] += g~_n(r; r_cut[si][sj]) Y_lm(r^) over the M neighbours given by their
   displacement vectors rij (x_j - x_i) and species sj; nu = sj*n_max + n                 */
static void env_A(const model_t *md, int si, int M, const double *rij, const int32_t *sj, double *A)
{
    int L2 = (md->l_max + 1) * (md->l_max + 1), Nv = md->S * md->n_max;
    double g[64], dg[64], Y[(LMAX_CAP + 1) * (LMAX_CAP + 1)];
    for (int a = 0; a < Nv * L2; a++) A[a] = 0.0;
    for (int j = 0; j < M; j++) {
        const double *d = rij + 3 * j;
        double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
        double u[3] = {d[0] / r, d[1] / r, d[2] / r};
        double rc = md->r_cut[si * md->S + sj[j]];
        oracle_radial(md->n_max, r, rc, g, dg);
        oracle_ylm(md->l_max, u, Y, NULL);
        for (int n = 0; n < md->n_max; n++)
            for (int lm = 0; lm < L2; lm++) A[(sj[j] * md->n_max + n) * L2 + lm] += g[n] * Y[lm];
    }
}

/* B[nu1<=nu2, l] = sum_m A[nu1,l,m] A[nu2,l,m] */
static void A_to_B(const model_t *md, const double *A, double *B)
{
    int L = md->l_max + 1, L2 = L * L, Nv = md->S * md->n_max;
    int p = 0;
    for (int v1 = 0; v1 < Nv; v1++)
        for (int v2 = v1; v2 < Nv; v2++)
            for (int l = 0; l < L; l++) {
                double s = 0.0;
                for (int m = -l; m <= l; m++) s += A[v1 * L2 + l * l + l + m] * A[v2 * L2 + l * l + l + m];
                B[p++] = s;
            }
}

/* Exported: descriptor of one explicit environment (used by the closed-form pins). */
int oracle_descriptor_env(int S, int n_max, int l_max, const double *r_cut, int si, int M, const double *rij,
                          const int32_t *sj, double *A, double *B, double *Bhat, double *nrm_out)
{
    model_t md = {S, n_max, l_max, r_cut, NULL, NULL};
    if (l_max > LMAX_CAP || n_max > 64 || S < 1) return ORACLE_ERR_ARG;
    int P = oracle_num_descriptors(S, n_max, l_max);
    env_A(&md, si, M, rij, sj, A);
    A_to_B(&md, A, B);
    double n2 = 0.0;
    for (int p = 0; p < P; p++) n2 += B[p] * B[p];
    double nrm = sqrt(n2);
    for (int p = 0; p < P; p++) Bhat[p] = (nrm > 0.0) ? B[p] / nrm : 0.0;
    *nrm_out = nrm;
    return ORACLE_OK;
}

/*
 * One atom: E_i (Eq. 1), V_i (Eq. 2) and g_ij = dE_i/dr_ij for each of its M neighbours,
 * by forming the gradient of the NORMALISED descriptor explicitly (the route P:L153 calls
 * "calculating forces directly from grad d_i"):
 *   dA[s_j,n,l,m]/dr_ij = g~_n'(r) Y_lm r^ + g~_n grad Y_lm,
 *   grad Y_lm = (1/r)(I - r^ r^T) grad_u Y~_lm(u)|_{u=r^}
 *   dB_p/dr   = sum_m (dA[nu1,l,m] A[nu2,l,m] + A[nu1,l,m] dA[nu2,l,m])
 *   dB^_p/dr  = dB_p/nrm - B^_p (sum_q B^_q dB_q)/nrm          (includes d nrm/dr: R11)
 *   dE/dr     = sum_p ((beta + beta^T) B^)_p dB^_p/dr
 * scratch must hold 4*Nv*L2 + 4*P doubles.
 */
static void atom_energy_grad(const model_t *md, int si, int M, const double *rij, const int32_t *sj, double *E,
                             double *V, double *g /* [M*3] or NULL */, double *scratch)
{
    int L = md->l_max + 1, L2 = L * L, Nv = md->S * md->n_max;
    int P = oracle_num_descriptors(md->S, md->n_max, md->l_max);
    double *A = scratch, *dA = A + Nv * L2, *B = dA + Nv * L2, *Bh = B + P, *bb = Bh + P, *dB = bb + P;
    const double *beta = md->beta + (size_t)si * P * P;
    *E = 0.0;
    if (V) *V = 0.0;
    if (g) for (int a = 0; a < 3 * M; a++) g[a] = 0.0;

    env_A(md, si, M, rij, sj, A);
    A_to_B(md, A, B);
    double n2 = 0.0;
    for (int p = 0; p < P; p++) n2 += B[p] * B[p];
    double nrm = sqrt(n2);
    if (!(nrm > 0.0)) return; /* empty neighbourhood (R8) */
    for (int p = 0; p < P; p++) Bh[p] = B[p] / nrm;

    double e = 0.0;
    for (int p = 0; p < P; p++) {
        double row = 0.0;
        for (int q = 0; q < P; q++) row += beta[(size_t)p * P + q] * Bh[q];
        e += Bh[p] * row;
    }
    *E = e;
    if (V && md->sigma) {
        const double *sg = md->sigma + (size_t)si * P * P;
        double v = 0.0;
        for (int p = 0; p < P; p++) {
            double row = 0.0;
            for (int q = 0; q < P; q++) row += sg[(size_t)p * P + q] * Bh[q];
            v += Bh[p] * row;
        }
        *V = v;
    }
    if (!g) return;

    /* bb = dE/dB^ = (beta + beta^T) B^ */
    for (int p = 0; p < P; p++) {
        double s = 0.0;
        for (int q = 0; q < P; q++) s += (beta[(size_t)p * P + q] + beta[(size_t)q * P + p]) * Bh[q];
        bb[p] = s;
    }
    double gr[64], dgr[64], Y[(LMAX_CAP + 1) * (LMAX_CAP + 1)], dY[3 * (LMAX_CAP + 1) * (LMAX_CAP + 1)];
    for (int j = 0; j < M; j++) {
        const double *d = rij + 3 * j;
        double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
        double u[3] = {d[0] / r, d[1] / r, d[2] / r};
        double rc = md->r_cut[si * md->S + sj[j]];
        oracle_radial(md->n_max, r, rc, gr, dgr);
        oracle_ylm(md->l_max, u, Y, dY);
        for (int dir = 0; dir < 3; dir++) {
            for (int a = 0; a < Nv * L2; a++) dA[a] = 0.0;
            for (int lm = 0; lm < L2; lm++) {
                double udY = u[0] * dY[3 * lm] + u[1] * dY[3 * lm + 1] + u[2] * dY[3 * lm + 2];
                double gY = (dY[3 * lm + dir] - u[dir] * udY) / r; /* tangential gradient of Y_lm */
                for (int n = 0; n < md->n_max; n++)
                    dA[(sj[j] * md->n_max + n) * L2 + lm] = dgr[n] * Y[lm] * u[dir] + gr[n] * gY;
            }
            int p = 0;
            for (int v1 = 0; v1 < Nv; v1++)
                for (int v2 = v1; v2 < Nv; v2++)
                    for (int l = 0; l < L; l++) {
                        double s = 0.0;
                        for (int m = -l; m <= l; m++) {
                            int k = l * l + l + m;
                            s += dA[v1 * L2 + k] * A[v2 * L2 + k] + A[v1 * L2 + k] * dA[v2 * L2 + k];
                        }
                        dB[p++] = s;
                    }
            double proj = 0.0;
            for (int q = 0; q < P; q++) proj += Bh[q] * dB[q];
            double acc = 0.0;
            for (int q = 0; q < P; q++) acc += bb[q] * (dB[q] / nrm - Bh[q] * proj / nrm);
            g[3 * j + dir] = acc;
        }
    }
}

static size_t scratch_doubles(const model_t *md)
{
    int L2 = (md->l_max + 1) * (md->l_max + 1), Nv = md->S * md->n_max;
    return (size_t)4 * Nv * L2 + (size_t)4 * oracle_num_descriptors(md->S, md->n_max, md->l_max) + 16;
}

/* gather displacement vectors and species of atom i's neighbours */
static void gather_env(const nlist_t *nl, int64_t i, const double *xw, const int32_t *types, const double box[9],
                       const int pbc[3], double *rij, int32_t *sj)
{
    int64_t m = nl->off[i + 1] - nl->off[i];
    for (int64_t q = 0; q < m; q++) {
        int64_t j = nl->idx[nl->off[i] + q];
        min_image(xw + 3 * i, xw + 3 * j, box, pbc, rij + 3 * q);
        sj[q] = types[j];
    }
}

/* Exported: A, B, B^, nrm of atom i of a whole system. */
int oracle_descriptor(int64_t N, const double *pos, const int32_t *types, const double box[9], const int pbc[3],
                      int S, int n_max, int l_max, const double *r_cut, int64_t i, double *A, double *B,
                      double *Bhat, double *nrm_out)
{
    int rc = check_system(box, pbc, S, r_cut);
    if (rc) return rc;
    if (i < 0 || i >= N) return ORACLE_ERR_ARG;
    double *xw = (double *)malloc(sizeof(double) * 3 * (size_t)N);
    oracle_wrap(N, pos, box, pbc, xw);
    nlist_t nl;
    rc = build_nlist(N, xw, types, box, pbc, S, r_cut, 1, &nl);
    if (rc == ORACLE_OK) {
        int64_t m = nl.off[i + 1] - nl.off[i];
        double *rij = (double *)malloc(sizeof(double) * 3 * (size_t)(m + 1));
        int32_t *sj = (int32_t *)malloc(sizeof(int32_t) * (size_t)(m + 1));
        gather_env(&nl, i, xw, types, box, pbc, rij, sj);
        rc = oracle_descriptor_env(S, n_max, l_max, r_cut, types[i], (int)m, rij, sj, A, B, Bhat, nrm_out);
        free(rij); free(sj);
    }
    nlist_free(&nl);
    free(xw);
    return rc;
}

/*
 * Exported: per-atom energies, forces and variances of the whole system (caller's order).
 *   F_i += g_ij,  F_j -= g_ij   with g_ij = dE_i/dr_ij, r_ij = x_j - x_i
 * e_out/f_out/v_out may each be NULL.  nbr_method: 0 brute force, 1 cell grid.
 */
static int compute_impl(int64_t N, const double *pos, const int32_t *types, const double box[9], const int pbc[3],
                        int S, int n_max, int l_max, const double *r_cut, const double *beta, const double *sigma,
                        int nbr_method, double *e_out, double *f_out, double *v_out, double *vir_out)
{
    model_t md = {S, n_max, l_max, r_cut, beta, sigma};
    int rc = check_system(box, pbc, S, r_cut);
    if (rc) return rc;
    if (l_max > LMAX_CAP || n_max > 64) return ORACLE_ERR_ARG;
    for (int64_t i = 0; i < N; i++) if (types[i] < 0 || types[i] >= S) return ORACLE_ERR_ARG;
    double *xw = (double *)malloc(sizeof(double) * 3 * (size_t)(N > 0 ? N : 1));
    if (!xw) return ORACLE_ERR_NOMEM;
    oracle_wrap(N, pos, box, pbc, xw);
    nlist_t nl;
    rc = build_nlist(N, xw, types, box, pbc, S, r_cut, nbr_method, &nl);
    if (rc) { free(xw); return rc; }
    int64_t npair = nl.off[N];
    double *gpair = (f_out || vir_out) ? (double *)malloc(sizeof(double) * 3 * (size_t)(npair > 0 ? npair : 1)) : NULL;
    int64_t mmax = 0;
    for (int64_t i = 0; i < N; i++) if (nl.off[i + 1] - nl.off[i] > mmax) mmax = nl.off[i + 1] - nl.off[i];

#ifdef _OPENMP
#pragma omp parallel
#endif
    {
        double *scratch = (double *)malloc(sizeof(double) * scratch_doubles(&md));
        double *rij = (double *)malloc(sizeof(double) * 3 * (size_t)(mmax + 1));
        int32_t *sj = (int32_t *)malloc(sizeof(int32_t) * (size_t)(mmax + 1));
#ifdef _OPENMP
#pragma omp for schedule(dynamic, 8)
#endif
        for (int64_t i = 0; i < N; i++) {
            int64_t m = nl.off[i + 1] - nl.off[i];
            double E, V;
            gather_env(&nl, i, xw, types, box, pbc, rij, sj);
            atom_energy_grad(&md, types[i], (int)m, rij, sj, &E, (v_out && sigma) ? &V : NULL,
                             gpair ? gpair + 3 * nl.off[i] : NULL, scratch);
            if (e_out) e_out[i] = E;
            if (v_out) v_out[i] = sigma ? V : 0.0;
        }
        free(scratch); free(rij); free(sj);
    }
    if (f_out) {
        for (int64_t a = 0; a < 3 * N; a++) f_out[a] = 0.0;
        for (int64_t i = 0; i < N; i++)
            for (int64_t q = nl.off[i]; q < nl.off[i + 1]; q++) {
                int64_t j = nl.idx[q];
                for (int d = 0; d < 3; d++) {
                    f_out[3 * i + d] += gpair[3 * q + d];
                    f_out[3 * j + d] -= gpair[3 * q + d];
                }
            }
    }
    if (vir_out) {
        /* Xi_ab = dE/d eps_ab under x -> (1 + eps) x: every r_ij -> (1 + eps) r_ij, so
           Xi_ab = sum_i sum_{j in N(i)} (dE_i/dr_ij)_a (r_ij)_b      (stress) */
        for (int a = 0; a < 9; a++) vir_out[a] = 0.0;
        for (int64_t i = 0; i < N; i++)
            for (int64_t q = nl.off[i]; q < nl.off[i + 1]; q++) {
                double d[3];
                min_image(xw + 3 * i, xw + 3 * nl.idx[q], box, pbc, d);
                for (int a = 0; a < 3; a++)
                    for (int b = 0; b < 3; b++) vir_out[3 * a + b] += gpair[3 * q + a] * d[b];
            }
    }
    free(gpair);
    nlist_free(&nl);
    free(xw);
    return ORACLE_OK;
}

int oracle_compute(int64_t N, const double *pos, const int32_t *types, const double box[9], const int pbc[3],
                   int S, int n_max, int l_max, const double *r_cut, const double *beta, const double *sigma,
                   int nbr_method, double *e_out, double *f_out, double *v_out)
{
    return compute_impl(N, pos, types, box, pbc, S, n_max, l_max, r_cut, beta, sigma, nbr_method, e_out, f_out, v_out,
                        NULL);
}

/* Exported: oracle_compute plus the virial Xi[3a+b] = dE/d eps_ab (eV); potential stress = Xi / volume. */
int oracle_compute_virial(int64_t N, const double *pos, const int32_t *types, const double box[9], const int pbc[3],
                          int S, int n_max, int l_max, const double *r_cut, const double *beta, const double *sigma,
                          int nbr_method, double *e_out, double *f_out, double *v_out, double *vir_out)
{
    return compute_impl(N, pos, types, box, pbc, S, n_max, l_max, r_cut, beta, sigma, nbr_method, e_out, f_out, v_out,
                        vir_out);
}

/*
 * Exported: the on-the-fly analysis of the paper's production run ("coordination numbers of H atoms ...
 * another H within 1 A"; "monitoring the maximum uncertainty"):
 *   max_unc = max_i sqrt(max(V_i, 0)); n_above = #{i : sqrt(max(V_i,0)) > threshold}
 *   coord[i] = #{j != i : s_j = species_b, |r_ij|^2 < r_coord^2 (minimum image)} if s_i = species_a, else 0
 * by brute force over all pairs.
 */
int oracle_analyze(int64_t N, const double *pos, const int32_t *types, const double box[9], const int pbc[3],
                   const double *var, double threshold, int species_a, int species_b, double r_coord,
                   double *max_unc, int64_t *n_above, int32_t *coord)
{
    if (!box_is_orthorhombic(box)) return ORACLE_ERR_BOX;
    double mx = 0.0;
    int64_t na = 0;
    if (var)
        for (int64_t i = 0; i < N; i++) {
            double u = sqrt(var[i] > 0.0 ? var[i] : 0.0);
            if (u > mx) mx = u;
            if (u > threshold) na++;
        }
    if (max_unc) *max_unc = mx;
    if (n_above) *n_above = na;
    if (coord) {
        double *xw = (double *)malloc(sizeof(double) * 3 * (size_t)(N > 0 ? N : 1));
        if (!xw) return ORACLE_ERR_NOMEM;
        oracle_wrap(N, pos, box, pbc, xw);
        for (int64_t i = 0; i < N; i++) {
            int32_t c = 0;
            if (types[i] == species_a)
                for (int64_t j = 0; j < N; j++) {
                    double d[3];
                    if (j == i || types[j] != species_b) continue;
                    min_image(xw + 3 * i, xw + 3 * j, box, pbc, d);
                    if (dist2(d) < r_coord * r_coord) c++;
                }
            coord[i] = c;
        }
        free(xw);
    }
    return ORACLE_OK;
}

/*
 * Exported: the same quantities for a SELECTION of atoms of a large system.
 * F_k needs dE_i/dx_k for i = k and every i with k in N(i), i.e. (symmetric cutoffs, R5)
 * i in {k} U N(k); each of those environments is evaluated in full.  Cell-grid neighbours.
 */
int oracle_compute_selected(int64_t N, const double *pos, const int32_t *types, const double box[9],
                            const int pbc[3], int S, int n_max, int l_max, const double *r_cut, const double *beta,
                            const double *sigma, int64_t n_sel, const int64_t *sel, int want_forces, double *e_out,
                            double *f_out, double *v_out)
{
    model_t md = {S, n_max, l_max, r_cut, beta, sigma};
    int rc = check_system(box, pbc, S, r_cut);
    if (rc) return rc;
    if (l_max > LMAX_CAP || n_max > 64) return ORACLE_ERR_ARG;
    double *xw = (double *)malloc(sizeof(double) * 3 * (size_t)(N > 0 ? N : 1));
    if (!xw) return ORACLE_ERR_NOMEM;
    oracle_wrap(N, pos, box, pbc, xw);
    nlist_t nl;
    rc = build_nlist(N, xw, types, box, pbc, S, r_cut, 1, &nl);
    if (rc) { free(xw); return rc; }
    int64_t mmax = 0;
    for (int64_t i = 0; i < N; i++) if (nl.off[i + 1] - nl.off[i] > mmax) mmax = nl.off[i + 1] - nl.off[i];

#ifdef _OPENMP
#pragma omp parallel
#endif
    {
        double *scratch = (double *)malloc(sizeof(double) * scratch_doubles(&md));
        double *rij = (double *)malloc(sizeof(double) * 3 * (size_t)(mmax + 1));
        double *g = (double *)malloc(sizeof(double) * 3 * (size_t)(mmax + 1));
        int32_t *sj = (int32_t *)malloc(sizeof(int32_t) * (size_t)(mmax + 1));
#ifdef _OPENMP
#pragma omp for schedule(dynamic, 1)
#endif
        for (int64_t t = 0; t < n_sel; t++) {
            int64_t k = sel[t];
            int64_t m = nl.off[k + 1] - nl.off[k];
            double E, V, F[3] = {0, 0, 0};
            gather_env(&nl, k, xw, types, box, pbc, rij, sj);
            atom_energy_grad(&md, types[k], (int)m, rij, sj, &E, (v_out && sigma) ? &V : NULL,
                             want_forces ? g : NULL, scratch);
            if (e_out) e_out[t] = E;
            if (v_out) v_out[t] = sigma ? V : 0.0;
            if (want_forces && f_out) {
                for (int64_t q = 0; q < m; q++)
                    for (int d = 0; d < 3; d++) F[d] += g[3 * q + d]; /* i = k term: F_k += g_kj */
                for (int64_t q = nl.off[k]; q < nl.off[k + 1]; q++) {
                    int64_t i = nl.idx[q]; /* i is a neighbour of k, so k is a neighbour of i */
                    int64_t mi = nl.off[i + 1] - nl.off[i];
                    double Ei;
                    gather_env(&nl, i, xw, types, box, pbc, rij, sj);
                    atom_energy_grad(&md, types[i], (int)mi, rij, sj, &Ei, NULL, g, scratch);
                    for (int64_t qq = 0; qq < mi; qq++)
                        if (nl.idx[nl.off[i] + qq] == k)
                            for (int d = 0; d < 3; d++) F[d] -= g[3 * qq + d]; /* F_k -= g_ik */
                }
                for (int d = 0; d < 3; d++) f_out[3 * t + d] = F[d];
            }
        }
        free(scratch); free(rij); free(g); free(sj);
    }
    nlist_free(&nl);
    free(xw);
    return ORACLE_OK;
}

/* ------------------------------------------------------------------ velocity Verlet (north_star; R12) */

/*
 * n_steps of: v += dt/2 kappa F/m ; x += dt v ; wrap ; F = F(x) ; v += dt/2 kappa F/m.
 * pos/vel are updated in place (pos left wrapped).  F(x0) is evaluated first.
 * pe_trace/ke_trace [n_steps+1]: sum_i E_i and sum 1/2 m v^2 / kappa after 0..n_steps steps.
 */
int oracle_step(int64_t N, double *pos, double *vel, const int32_t *types, const double *mass /*[S]*/,
                const double box[9], const int pbc[3], int S, int n_max, int l_max, const double *r_cut,
                const double *beta, const double *sigma, int nbr_method, double dt, int n_steps, double *e_out,
                double *f_out, double *v_out, double *pe_trace, double *ke_trace)
{
    double *E = (double *)malloc(sizeof(double) * (size_t)(N > 0 ? N : 1));
    double *F = (double *)malloc(sizeof(double) * 3 * (size_t)(N > 0 ? N : 1));
    double *V = (double *)malloc(sizeof(double) * (size_t)(N > 0 ? N : 1));
    if (!E || !F || !V) return ORACLE_ERR_NOMEM;
    oracle_wrap(N, pos, box, pbc, pos);
    int rc = oracle_compute(N, pos, types, box, pbc, S, n_max, l_max, r_cut, beta, sigma, nbr_method, E, F, V);
    for (int step = 0; rc == ORACLE_OK && step <= n_steps; step++) {
        double pe = 0.0, ke = 0.0;
        for (int64_t i = 0; i < N; i++) {
            pe += E[i];
            for (int d = 0; d < 3; d++) ke += 0.5 * mass[types[i]] * vel[3 * i + d] * vel[3 * i + d] / KAPPA;
        }
        if (pe_trace) pe_trace[step] = pe;
        if (ke_trace) ke_trace[step] = ke;
        if (step == n_steps) break;
        for (int64_t i = 0; i < N; i++)
            for (int d = 0; d < 3; d++) {
                vel[3 * i + d] += 0.5 * dt * KAPPA * F[3 * i + d] / mass[types[i]];
                pos[3 * i + d] += dt * vel[3 * i + d];
            }
        oracle_wrap(N, pos, box, pbc, pos);
        rc = oracle_compute(N, pos, types, box, pbc, S, n_max, l_max, r_cut, beta, sigma, nbr_method, E, F, V);
        if (rc) break;
        for (int64_t i = 0; i < N; i++)
            for (int d = 0; d < 3; d++) vel[3 * i + d] += 0.5 * dt * KAPPA * F[3 * i + d] / mass[types[i]];
    }
    if (e_out) memcpy(e_out, E, sizeof(double) * (size_t)N);
    if (f_out) memcpy(f_out, F, sizeof(double) * 3 * (size_t)N);
    if (v_out) memcpy(v_out, V, sizeof(double) * (size_t)N);
    free(E); free(F); free(V);
    return rc;
}

/* ------------------------------------------------------------------ Nose-Hoover NVT (R19) */

#define KB_EV 8.617333262e-5 /* eV/K (R13) */

/* half step of the single Nose-Hoover thermostat (Martyna-Tuckerman-Klein splitting), h = dt/2:
 *   xi += (h/2)(K2 - g kT)/Q ;  v *= exp(-xi h) ;  eta += xi h ;  xi += (h/2)(K2' - g kT)/Q
 * with K2 = sum m v^2 / kappa (twice the kinetic energy, eV), Q = g kT tau^2, g = 3N - 3. */
static void nh_half(int64_t N, double *vel, const int32_t *types, const double *mass, double h, double gkT, double Q,
                    double *xi, double *eta)
{
    double K2 = 0.0;
    for (int64_t i = 0; i < N; i++)
        for (int d = 0; d < 3; d++) K2 += mass[types[i]] * vel[3 * i + d] * vel[3 * i + d] / KAPPA;
    *xi += 0.5 * h * (K2 - gkT) / Q;
    double s = exp(-(*xi) * h);
    for (int64_t a = 0; a < 3 * N; a++) vel[a] *= s;
    K2 *= s * s;
    *eta += (*xi) * h;
    *xi += 0.5 * h * (K2 - gkT) / Q;
}

/*
 * n_steps of: thermostat half step ; velocity Verlet (as oracle_step) ; thermostat half step.
 * xi_eta[2] = {xi (1/fs), eta} is read and updated.  cons_trace [n_steps+1]: the conserved quantity
 * KE + PE + Q xi^2 / 2 + g kT eta after 0..n_steps steps; temp_trace: 2 KE / (g k_B).
 */
int oracle_step_nvt(int64_t N, double *pos, double *vel, const int32_t *types, const double *mass,
                    const double box[9], const int pbc[3], int S, int n_max, int l_max, const double *r_cut,
                    const double *beta, const double *sigma, int nbr_method, double dt, int n_steps, double T_target,
                    double tau, double *xi_eta, double *e_out, double *f_out, double *cons_trace, double *temp_trace)
{
    if (N < 2 || !(T_target > 0.0) || !(tau > 0.0)) return ORACLE_ERR_ARG;
    double *E = (double *)malloc(sizeof(double) * (size_t)N);
    double *F = (double *)malloc(sizeof(double) * 3 * (size_t)N);
    if (!E || !F) return ORACLE_ERR_NOMEM;
    const double g = 3.0 * (double)N - 3.0;
    const double gkT = g * KB_EV * T_target;
    const double Q = gkT * tau * tau;
    double xi = xi_eta[0], eta = xi_eta[1];
    oracle_wrap(N, pos, box, pbc, pos);
    int rc = oracle_compute(N, pos, types, box, pbc, S, n_max, l_max, r_cut, beta, sigma, nbr_method, E, F, NULL);
    for (int step = 0; rc == ORACLE_OK && step <= n_steps; step++) {
        double pe = 0.0, ke = 0.0;
        for (int64_t i = 0; i < N; i++) {
            pe += E[i];
            for (int d = 0; d < 3; d++) ke += 0.5 * mass[types[i]] * vel[3 * i + d] * vel[3 * i + d] / KAPPA;
        }
        if (cons_trace) cons_trace[step] = ke + pe + 0.5 * Q * xi * xi + gkT * eta;
        if (temp_trace) temp_trace[step] = 2.0 * ke / (g * KB_EV);
        if (step == n_steps) break;
        nh_half(N, vel, types, mass, 0.5 * dt, gkT, Q, &xi, &eta);
        for (int64_t i = 0; i < N; i++)
            for (int d = 0; d < 3; d++) {
                vel[3 * i + d] += 0.5 * dt * KAPPA * F[3 * i + d] / mass[types[i]];
                pos[3 * i + d] += dt * vel[3 * i + d];
            }
        oracle_wrap(N, pos, box, pbc, pos);
        rc = oracle_compute(N, pos, types, box, pbc, S, n_max, l_max, r_cut, beta, sigma, nbr_method, E, F, NULL);
        if (rc) break;
        for (int64_t i = 0; i < N; i++)
            for (int d = 0; d < 3; d++) vel[3 * i + d] += 0.5 * dt * KAPPA * F[3 * i + d] / mass[types[i]];
        nh_half(N, vel, types, mass, 0.5 * dt, gkT, Q, &xi, &eta);
    }
    xi_eta[0] = xi;
    xi_eta[1] = eta;
    if (e_out) memcpy(e_out, E, sizeof(double) * (size_t)N);
    if (f_out) memcpy(f_out, F, sizeof(double) * 3 * (size_t)N);
    free(E); free(F);
    return rc;
}
