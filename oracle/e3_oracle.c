/*
 * e3_oracle.c -- fp64 CPU ORACLE for the e3j hot path.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * leg may call this.  It shares no code, header, table or constant with the CUDA path
 * under paper_2605_22698_b200/ and must never be used by the product path.
 *
 * What it is: the plain definition of every step of the hot path, written as dense
 * loops in double precision, in the order and notation of SURVEY.md section 8(c)
 * (the paper, arxiv 2605.22698, only *names* the operation -- PAPER.md L72-L74
 * "Clebsch-Gordan Tensor Product", L66 "edge vectors from stored positions and
 * connectivity", L82 "fusion of the message passing kernel" -- and gives no formula;
 * the textbook definitions used here are the readings A1..A18 listed in DESIGN.md).
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): every function below is pinned
 * against something that is not itself -- explicit low-order polynomials, the
 * addition theorem, a library complex SH, CG closed forms and orthogonality, the
 * Gaunt-type SH<->CG identity, Wigner-D equivariance, textbook special cases
 * (adjacency SpMV, dot and cross products), finite differences, the Euler identity
 * of the trilinear map, momentum/torque conservation and numpy's stable argsort.
 * Nothing here is "parity unpinned".
 *
 * Layouts (reading A7): a node row is the concatenation of its irrep blocks; inside a
 * block the index is m*C + u (channel fastest).  SH row index l*l + l + m.  Weights
 * [(e*P + p)*C + u].  All floating inputs/outputs are double; all indices int32.
 *
 * Threading: `#pragma omp parallel for` only over loops whose iterations write
 * disjoint outputs (receivers for out, senders for dx, edges for dY/dw), so every
 * output element is summed in ascending edge order exactly as in a serial loop.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct { int l; int parity; int mul; } orc_irrep;
typedef struct { int i_in; int l_sh; int i_out; } orc_path;

#define ORC_LMAX 8

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void orc_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

static double fact(int n)
{
    double f = 1.0;
    for (int i = 2; i <= n; ++i) f *= (double)i;
    return f;
}

/* ------------------------------------------------------------------------------------
 * Clebsch-Gordan coefficients.
 * Reading A4 (PAPER.md L44 cites the CG formalism without fixing a convention):
 * Condon-Shortley complex coefficient <l1 m1 l2 m2 | l3 m3> from Racah's closed form
 *   delta(m3, m1+m2) * sqrt[(2l3+1) (l3+l1-l2)! (l3-l1+l2)! (l1+l2-l3)! / (l1+l2+l3+1)!]
 *   * sqrt[(l3+m3)! (l3-m3)! (l1-m1)! (l1+m1)! (l2-m2)! (l2+m2)!]
 *   * sum_k (-1)^k / [k! (l1+l2-l3-k)! (l1-m1-k)! (l2+m2-k)! (l3-l2+m1+k)! (l3-l1-m2+k)!]
 * ---------------------------------------------------------------------------------- */
double orc_cg_complex(int l1, int m1, int l2, int m2, int l3, int m3)
{
    if (m1 + m2 != m3) return 0.0;
    if (l3 < abs(l1 - l2) || l3 > l1 + l2) return 0.0;
    if (abs(m1) > l1 || abs(m2) > l2 || abs(m3) > l3) return 0.0;
    double pref = sqrt((2.0 * l3 + 1.0) * fact(l3 + l1 - l2) * fact(l3 - l1 + l2) * fact(l1 + l2 - l3)
                       / fact(l1 + l2 + l3 + 1));
    pref *= sqrt(fact(l3 + m3) * fact(l3 - m3) * fact(l1 - m1) * fact(l1 + m1) * fact(l2 - m2) * fact(l2 + m2));
    double sum = 0.0;
    for (int k = 0; k <= l1 + l2 + l3; ++k) {
        int a0 = k, a1 = l1 + l2 - l3 - k, a2 = l1 - m1 - k, a3 = l2 + m2 - k;
        int a4 = l3 - l2 + m1 + k, a5 = l3 - l1 - m2 + k;
        if (a0 < 0 || a1 < 0 || a2 < 0 || a3 < 0 || a4 < 0 || a5 < 0) continue;
        double den = fact(a0) * fact(a1) * fact(a2) * fact(a3) * fact(a4) * fact(a5);
        sum += ((k & 1) ? -1.0 : 1.0) / den;
    }
    return pref * sum;
}

/* Reading A1: unitary change of basis complex(CS) -> real, Y^real_m = sum_mu U[m,mu] Y^complex_mu.
 *   U[0,0] = 1
 *   m > 0:          U[m,-m] = 1/sqrt2,   U[m,m]  = (-1)^m / sqrt2        (cos-type)
 *   m < 0, a = |m|: U[m,-a] = i/sqrt2,   U[m,a]  = -i (-1)^a / sqrt2     (sin-type)
 * Stored as U[(m+l)*(2l+1) + (mu+l)]. */
static void real_basis_U(int l, double complex *U)
{
    int d = 2 * l + 1;
    for (int i = 0; i < d * d; ++i) U[i] = 0.0;
    const double s = 1.0 / sqrt(2.0);
    for (int m = -l; m <= l; ++m) {
        if (m == 0) {
            U[l * d + l] = 1.0;
        } else if (m > 0) {
            U[(m + l) * d + (-m + l)] = s;
            U[(m + l) * d + (m + l)] = ((m & 1) ? -1.0 : 1.0) * s;
        } else {
            int a = -m;
            U[(m + l) * d + (-a + l)] = I * s;
            U[(m + l) * d + (a + l)] = -I * ((a & 1) ? -1.0 : 1.0) * s;
        }
    }
}

/* Reading A4: real CG tensor, dense, C[(m1+l1)*(2l2+1)*(2l3+1) + (m2+l2)*(2l3+1) + (m3+l3)]
 *   T = sum_{mu1,mu2,mu3} U1[m1,mu1] U2[m2,mu2] conj(U3[m3,mu3]) <l1 mu1 l2 mu2 | l3 mu3>
 * T is purely real when l1+l2+l3 is even (C = Re T) and purely imaginary when odd
 * (C = Im T).  Returns max |discarded part| so the caller can check that claim. */
double orc_cg_real(int l1, int l2, int l3, double *C)
{
    int d1 = 2 * l1 + 1, d2 = 2 * l2 + 1, d3 = 2 * l3 + 1;
    double complex U1[(2 * ORC_LMAX + 1) * (2 * ORC_LMAX + 1)];
    double complex U2[(2 * ORC_LMAX + 1) * (2 * ORC_LMAX + 1)];
    double complex U3[(2 * ORC_LMAX + 1) * (2 * ORC_LMAX + 1)];
    real_basis_U(l1, U1);
    real_basis_U(l2, U2);
    real_basis_U(l3, U3);
    int odd = (l1 + l2 + l3) & 1;
    double discarded = 0.0;
    for (int m1 = -l1; m1 <= l1; ++m1)
        for (int m2 = -l2; m2 <= l2; ++m2)
            for (int m3 = -l3; m3 <= l3; ++m3) {
                double complex T = 0.0;
                for (int u1 = -l1; u1 <= l1; ++u1)
                    for (int u2 = -l2; u2 <= l2; ++u2)
                        for (int u3 = -l3; u3 <= l3; ++u3) {
                            double c = orc_cg_complex(l1, u1, l2, u2, l3, u3);
                            if (c == 0.0) continue;
                            T += U1[(m1 + l1) * d1 + (u1 + l1)] * U2[(m2 + l2) * d2 + (u2 + l2)]
                                 * conj(U3[(m3 + l3) * d3 + (u3 + l3)]) * c;
                        }
                double keep = odd ? cimag(T) : creal(T);
                double drop = odd ? creal(T) : cimag(T);
                if (fabs(drop) > discarded) discarded = fabs(drop);
                C[((m1 + l1) * d2 + (m2 + l2)) * d3 + (m3 + l3)] = keep;
            }
    return discarded;
}

/* ------------------------------------------------------------------------------------
 * Real spherical harmonics, component normalisation (readings A1, A2, A3).
 * Complex SH with Condon-Shortley phase, written on the unit vector (x,y,z):
 *   Y_l^m = (-1)^m sqrt[(2l+1)/(4 pi) (l-m)!/(l+m)!] (d^m P_l/dz^m)(z) (x+iy)^m ,  m >= 0
 *   Y_l^{-m} = (-1)^m conj(Y_l^m)
 * ((1-z^2)^{m/2} e^{i m phi} = (x+iy)^m on the unit sphere), Legendre polynomial
 *   P_l(z) = 2^-l sum_k (-1)^k binom(l,k) binom(2l-2k,l) z^(l-2k).
 * Real SH = U_l . Y^complex, times sqrt(4 pi) ("component" normalisation,
 * sum_m Y_lm^2 = 2l+1).
 * ---------------------------------------------------------------------------------- */
static double binom(int n, int k)
{
    return fact(n) / (fact(k) * fact(n - k));
}

/* value of d^m P_l / dz^m (order = m) or its next derivative (order = m+1) at z */
static double legendre_deriv(int l, int order, double z)
{
    double s = 0.0;
    for (int k = 0; 2 * k <= l; ++k) {
        int p = l - 2 * k;
        if (p < order) continue;
        double c = ((k & 1) ? -1.0 : 1.0) * binom(l, k) * binom(2 * l - 2 * k, l) / pow(2.0, l);
        c *= fact(p) / fact(p - order);
        s += c * pow(z, p - order);
    }
    return s;
}

static double complex cpow_int(double complex a, int n)
{
    double complex r = 1.0;
    for (int i = 0; i < n; ++i) r *= a;
    return r;
}

/* complex SH of degree l on unit vector u, and (if gradF != NULL) the Cartesian
 * gradient of its polynomial extension F(x,y,z) = N Q(z) (x+iy)^m, both times sqrt(4 pi) */
static void complex_sh_unit(int l, const double u[3], double complex *Yc, double complex (*gradF)[3])
{
    double x = u[0], y = u[1], z = u[2];
    double complex xi = x + I * y;
    for (int m = 0; m <= l; ++m) {
        double N = ((m & 1) ? -1.0 : 1.0) * sqrt((2.0 * l + 1.0) * fact(l - m) / fact(l + m));
        double Q = legendre_deriv(l, m, z);
        double dQ = legendre_deriv(l, m + 1, z);
        double complex xm = cpow_int(xi, m);
        double complex xm1 = (m > 0) ? cpow_int(xi, m - 1) : 0.0;
        double complex val = N * Q * xm;
        double complex gx = N * Q * (double)m * xm1;
        double complex gy = N * Q * (double)m * xm1 * I;
        double complex gz = N * dQ * xm;
        double sgn = (m & 1) ? -1.0 : 1.0;
        Yc[m + l] = val;
        Yc[-m + l] = sgn * conj(val);
        if (gradF) {
            gradF[m + l][0] = gx; gradF[m + l][1] = gy; gradF[m + l][2] = gz;
            gradF[-m + l][0] = sgn * conj(gx); gradF[-m + l][1] = sgn * conj(gy); gradF[-m + l][2] = sgn * conj(gz);
        }
    }
}

/* Y[n, (lmax+1)^2] from raw (un-normalised) vectors vec[n,3].
 * A3: |r| == 0 exactly -> r^ := 0, so Y_00 = 1 and Y_{l>0} = 0. */
void orc_sh(int lmax, int64_t n, const double *vec, double *Y)
{
    int sh_dim = (lmax + 1) * (lmax + 1);
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < n; ++e) {
        const double *r = vec + 3 * e;
        double *Ye = Y + (int64_t)sh_dim * e;
        double nr = sqrt(r[0] * r[0] + r[1] * r[1] + r[2] * r[2]);
        if (nr == 0.0) {
            for (int i = 0; i < sh_dim; ++i) Ye[i] = 0.0;
            Ye[0] = 1.0;
            continue;
        }
        double u[3] = { r[0] / nr, r[1] / nr, r[2] / nr };
        for (int l = 0; l <= lmax; ++l) {
            int d = 2 * l + 1;
            double complex Yc[2 * ORC_LMAX + 1];
            double complex U[(2 * ORC_LMAX + 1) * (2 * ORC_LMAX + 1)];
            complex_sh_unit(l, u, Yc, NULL);
            real_basis_U(l, U);
            for (int m = -l; m <= l; ++m) {
                double complex s = 0.0;
                for (int mu = -l; mu <= l; ++mu) s += U[(m + l) * d + (mu + l)] * Yc[mu + l];
                Ye[l * l + l + m] = creal(s);
            }
        }
    }
}

/* Jacobian J[n, sh_dim, 3] = d Y_lm(r/|r|) / d r.
 * Chain rule through the normalisation:
 *   dY/dr = (1/|r|) (I - r^ r^T) grad F_lm(r^),  F_lm the polynomial extension above.
 * A3: zero vector -> zero Jacobian. */
void orc_sh_jac(int lmax, int64_t n, const double *vec, double *J)
{
    int sh_dim = (lmax + 1) * (lmax + 1);
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < n; ++e) {
        const double *r = vec + 3 * e;
        double *Je = J + (int64_t)sh_dim * 3 * e;
        double nr = sqrt(r[0] * r[0] + r[1] * r[1] + r[2] * r[2]);
        if (nr == 0.0) {
            for (int i = 0; i < sh_dim * 3; ++i) Je[i] = 0.0;
            continue;
        }
        double u[3] = { r[0] / nr, r[1] / nr, r[2] / nr };
        for (int l = 0; l <= lmax; ++l) {
            int d = 2 * l + 1;
            double complex Yc[2 * ORC_LMAX + 1];
            double complex G[2 * ORC_LMAX + 1][3];
            double complex U[(2 * ORC_LMAX + 1) * (2 * ORC_LMAX + 1)];
            complex_sh_unit(l, u, Yc, G);
            real_basis_U(l, U);
            for (int m = -l; m <= l; ++m) {
                double g[3];
                for (int a = 0; a < 3; ++a) {
                    double complex s = 0.0;
                    for (int mu = -l; mu <= l; ++mu) s += U[(m + l) * d + (mu + l)] * G[mu + l][a];
                    g[a] = creal(s);
                }
                double gu = g[0] * u[0] + g[1] * u[1] + g[2] * u[2];
                for (int a = 0; a < 3; ++a) Je[(l * l + l + m) * 3 + a] = (g[a] - u[a] * gu) / nr;
            }
        }
    }
}

/* dvec[e,:] = sum_lm dY[e,lm] * dY_lm/dr */
void orc_sh_bwd(int lmax, int64_t n, const double *vec, const double *dY, double *dvec)
{
    int sh_dim = (lmax + 1) * (lmax + 1);
    double *J = (double *)malloc(sizeof(double) * (size_t)n * sh_dim * 3);
    orc_sh_jac(lmax, n, vec, J);
    for (int64_t e = 0; e < n; ++e)
        for (int a = 0; a < 3; ++a) {
            double s = 0.0;
            for (int i = 0; i < sh_dim; ++i) s += dY[e * sh_dim + i] * J[(e * sh_dim + i) * 3 + a];
            dvec[3 * e + a] = s;
        }
    free(J);
}

/* ------------------------------------------------------------------------------------
 * Graph preparation: CSR over receivers, stable sender-sorted
 * permutation and CSC-style pointer.  Integer only.
 *   row_ptr[r] = #edges with receiver < r ;  col_ptr[s] = #edges with sender < s ;
 *   perm_s = edge ids ordered by sender, ties in ascending edge id (stable).
 * ---------------------------------------------------------------------------------- */
int orc_graph_prepare(const int32_t *senders, const int32_t *receivers, int64_t E, int32_t N,
                      int32_t *row_ptr, int32_t *perm_s, int32_t *col_ptr)
{
    for (int32_t i = 0; i <= N; ++i) { row_ptr[i] = 0; col_ptr[i] = 0; }
    for (int64_t e = 0; e < E; ++e) {
        if (receivers[e] < 0 || receivers[e] >= N || senders[e] < 0 || senders[e] >= N) return 1;
        row_ptr[receivers[e] + 1] += 1;
        col_ptr[senders[e] + 1] += 1;
    }
    for (int32_t i = 0; i < N; ++i) { row_ptr[i + 1] += row_ptr[i]; col_ptr[i + 1] += col_ptr[i]; }
    int32_t *fill = (int32_t *)malloc(sizeof(int32_t) * (size_t)(N + 1));
    memcpy(fill, col_ptr, sizeof(int32_t) * (size_t)(N + 1));
    for (int64_t e = 0; e < E; ++e) perm_s[fill[senders[e]]++] = (int32_t)e;
    free(fill);
    return 0;
}

/* stable grouping of edge ids by key (receiver or sender); ptr[N+1], list[E] */
static void group_edges(const int32_t *key, int64_t E, int32_t N, int64_t *ptr, int64_t *list)
{
    for (int32_t i = 0; i <= N; ++i) ptr[i] = 0;
    for (int64_t e = 0; e < E; ++e) ptr[key[e] + 1] += 1;
    for (int32_t i = 0; i < N; ++i) ptr[i + 1] += ptr[i];
    int64_t *fill = (int64_t *)malloc(sizeof(int64_t) * (size_t)(N + 1));
    memcpy(fill, ptr, sizeof(int64_t) * (size_t)(N + 1));
    for (int64_t e = 0; e < E; ++e) list[fill[key[e]]++] = e;
    free(fill);
}

/* block offsets (in units of C-wide rows) of each irrep inside a node row */
static int block_offsets(const orc_irrep *ir, int n, int *off)
{
    int o = 0;
    for (int i = 0; i < n; ++i) { off[i] = o; o += 2 * ir[i].l + 1; }
    return o;
}

typedef struct {
    int n_paths, C, in_dim, out_dim, sh_dim;
    int l1[256], l2[256], l3[256], in_off[256], out_off[256];
    double *cg[256]; /* dense real CG tensor of each path */
} orc_plan;

/* Validates the path table (triangle + parity rules, reading A5) and builds dense CG tensors. */
static int plan_build(orc_plan *pl, const orc_irrep *irreps_in, int n_in, int sh_lmax,
                      const orc_irrep *irreps_out, int n_out, const orc_path *paths, int n_paths)
{
    int in_off[256], out_off[256];
    pl->n_paths = 0;
    if (n_paths > 256 || n_in > 256 || n_out > 256 || n_in < 1 || n_out < 1) return 1;
    for (int p = 0; p < n_paths; ++p) pl->cg[p] = NULL;
    pl->in_dim = block_offsets(irreps_in, n_in, in_off);
    pl->out_dim = block_offsets(irreps_out, n_out, out_off);
    pl->sh_dim = (sh_lmax + 1) * (sh_lmax + 1);
    pl->C = irreps_in[0].mul;
    for (int i = 0; i < n_in; ++i) if (irreps_in[i].mul != pl->C) return 2;
    for (int i = 0; i < n_out; ++i) if (irreps_out[i].mul != pl->C) return 2;
    pl->n_paths = n_paths;
    for (int p = 0; p < n_paths; ++p) {
        orc_path q = paths[p];
        if (q.i_in < 0 || q.i_in >= n_in || q.i_out < 0 || q.i_out >= n_out) return 3;
        if (q.l_sh < 0 || q.l_sh > sh_lmax) return 3;
        int l1 = irreps_in[q.i_in].l, l2 = q.l_sh, l3 = irreps_out[q.i_out].l;
        if (l3 < abs(l1 - l2) || l3 > l1 + l2) return 4;                          /* triangle rule */
        int par = irreps_in[q.i_in].parity * ((l2 & 1) ? -1 : 1);                  /* Y_l has parity (-1)^l */
        if (par != irreps_out[q.i_out].parity) return 5;                           /* parity rule */
        pl->l1[p] = l1; pl->l2[p] = l2; pl->l3[p] = l3;
        pl->in_off[p] = in_off[q.i_in]; pl->out_off[p] = out_off[q.i_out];
        pl->cg[p] = (double *)malloc(sizeof(double) * (size_t)((2 * l1 + 1) * (2 * l2 + 1) * (2 * l3 + 1)));
        orc_cg_real(l1, l2, l3, pl->cg[p]);
    }
    return 0;
}

static void plan_free(orc_plan *pl)
{
    for (int p = 0; p < pl->n_paths; ++p) free(pl->cg[p]);
}

int orc_plan_dims(const orc_irrep *irreps_in, int n_in, int sh_lmax, const orc_irrep *irreps_out, int n_out,
                  const orc_path *paths, int n_paths, int *in_dim, int *sh_dim, int *out_dim)
{
    orc_plan pl;
    int rc = plan_build(&pl, irreps_in, n_in, sh_lmax, irreps_out, n_out, paths, n_paths);
    if (rc) { plan_free(&pl); return rc; }
    *in_dim = pl.in_dim; *sh_dim = pl.sh_dim; *out_dim = pl.out_dim;
    plan_free(&pl);
    return 0;
}

/* ------------------------------------------------------------------------------------
 * Fused gather - tensor product - scatter, forward:
 *   out[r, blk(p), m3, u] = sum_{e in in(r)} w[e,p,u] *
 *        sum_{m1,m2} C^p[m1,m2,m3] * x[snd(e), blk(l1(p)), m1, u] * Y[e, l2(p), m2]
 * Paths that name the same i_out add (reading A6).  Every out row is written (zeros
 * for isolated receivers, A11).  Edges may come in any order.
 * ---------------------------------------------------------------------------------- */
int orc_tp_scatter_fwd(const orc_irrep *irreps_in, int n_in, int sh_lmax, const orc_irrep *irreps_out, int n_out,
                       const orc_path *paths, int n_paths,
                       const double *x, const double *sh, const double *w,
                       const int32_t *senders, const int32_t *receivers, int64_t E, int32_t N, double *out)
{
    orc_plan pl;
    int rc = plan_build(&pl, irreps_in, n_in, sh_lmax, irreps_out, n_out, paths, n_paths);
    if (rc) { plan_free(&pl); return rc; }
    const int C = pl.C, P = pl.n_paths;
    int64_t *ptr = (int64_t *)malloc(sizeof(int64_t) * (size_t)(N + 1));
    int64_t *list = (int64_t *)malloc(sizeof(int64_t) * (size_t)(E > 0 ? E : 1));
    group_edges(receivers, E, N, ptr, list);
#pragma omp parallel for schedule(dynamic, 8)
    for (int32_t r = 0; r < N; ++r) {
        double *o = out + (int64_t)r * pl.out_dim * C;
        for (int i = 0; i < pl.out_dim * C; ++i) o[i] = 0.0;
        for (int64_t j = ptr[r]; j < ptr[r + 1]; ++j) {
            int64_t e = list[j];
            const double *xs = x + (int64_t)senders[e] * pl.in_dim * C;
            const double *Ye = sh + e * pl.sh_dim;
            for (int p = 0; p < P; ++p) {
                int l1 = pl.l1[p], l2 = pl.l2[p], l3 = pl.l3[p];
                int d2 = 2 * l2 + 1, d3 = 2 * l3 + 1;
                const double *Cp = pl.cg[p];
                const double *wp = w + (e * P + p) * C;
                for (int m1 = 0; m1 <= 2 * l1; ++m1)
                    for (int m2 = 0; m2 <= 2 * l2; ++m2)
                        for (int m3 = 0; m3 <= 2 * l3; ++m3) {
                            double c = Cp[(m1 * d2 + m2) * d3 + m3];
                            if (c == 0.0) continue;
                            double cy = c * Ye[l2 * l2 + m2];
                            const double *xb = xs + (pl.in_off[p] + m1) * C;
                            double *ob = o + (pl.out_off[p] + m3) * C;
                            for (int u = 0; u < C; ++u) ob[u] += wp[u] * cy * xb[u];
                        }
            }
        }
    }
    free(ptr); free(list);
    plan_free(&pl);
    return 0;
}

/* ------------------------------------------------------------------------------------
 * VJP of the forward.  Given g = dL/d out:
 *   dx[s,l1,m1,u] = sum_{e in out(s)} sum_p w[e,p,u] sum_{m2,m3} C^p Y[e,l2,m2] g[rcv(e),p,m3,u]
 *   dY[e,l2,m2]   = sum_p sum_u w[e,p,u] sum_{m1,m3} C^p x[s,l1,m1,u] g[r,p,m3,u]
 *   dw[e,p,u]     = sum_{m1,m2,m3} C^p x[s,l1,m1,u] Y[e,l2,m2] g[r,p,m3,u]
 * ---------------------------------------------------------------------------------- */
int orc_tp_scatter_bwd(const orc_irrep *irreps_in, int n_in, int sh_lmax, const orc_irrep *irreps_out, int n_out,
                       const orc_path *paths, int n_paths,
                       const double *x, const double *sh, const double *w,
                       const int32_t *senders, const int32_t *receivers, int64_t E, int32_t N,
                       const double *g, double *dx, double *dY, double *dw)
{
    orc_plan pl;
    int rc = plan_build(&pl, irreps_in, n_in, sh_lmax, irreps_out, n_out, paths, n_paths);
    if (rc) { plan_free(&pl); return rc; }
    const int C = pl.C, P = pl.n_paths;

    /* dY and dw: one independent result per edge */
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t e = 0; e < E; ++e) {
        const double *xs = x + (int64_t)senders[e] * pl.in_dim * C;
        const double *gr = g + (int64_t)receivers[e] * pl.out_dim * C;
        const double *Ye = sh + e * pl.sh_dim;
        double *dYe = dY + e * pl.sh_dim;
        for (int i = 0; i < pl.sh_dim; ++i) dYe[i] = 0.0;
        for (int p = 0; p < P; ++p) {
            int l1 = pl.l1[p], l2 = pl.l2[p], l3 = pl.l3[p];
            int d2 = 2 * l2 + 1, d3 = 2 * l3 + 1;
            const double *Cp = pl.cg[p];
            const double *wp = w + (e * P + p) * C;
            double *dwp = dw + (e * P + p) * C;
            for (int u = 0; u < C; ++u) dwp[u] = 0.0;
            for (int m1 = 0; m1 <= 2 * l1; ++m1)
                for (int m2 = 0; m2 <= 2 * l2; ++m2)
                    for (int m3 = 0; m3 <= 2 * l3; ++m3) {
                        double c = Cp[(m1 * d2 + m2) * d3 + m3];
                        if (c == 0.0) continue;
                        const double *xb = xs + (pl.in_off[p] + m1) * C;
                        const double *gb = gr + (pl.out_off[p] + m3) * C;
                        double y = Ye[l2 * l2 + m2];
                        double acc = 0.0;
                        for (int u = 0; u < C; ++u) {
                            double xg = c * xb[u] * gb[u];
                            dwp[u] += xg * y;
                            acc += wp[u] * xg;
                        }
                        dYe[l2 * l2 + m2] += acc;
                    }
        }
    }

    /* dx: sum over the out-edges of each sender, ascending edge id */
    int64_t *ptr = (int64_t *)malloc(sizeof(int64_t) * (size_t)(N + 1));
    int64_t *list = (int64_t *)malloc(sizeof(int64_t) * (size_t)(E > 0 ? E : 1));
    group_edges(senders, E, N, ptr, list);
#pragma omp parallel for schedule(dynamic, 8)
    for (int32_t s = 0; s < N; ++s) {
        double *d = dx + (int64_t)s * pl.in_dim * C;
        for (int i = 0; i < pl.in_dim * C; ++i) d[i] = 0.0;
        for (int64_t j = ptr[s]; j < ptr[s + 1]; ++j) {
            int64_t e = list[j];
            const double *gr = g + (int64_t)receivers[e] * pl.out_dim * C;
            const double *Ye = sh + e * pl.sh_dim;
            for (int p = 0; p < P; ++p) {
                int l1 = pl.l1[p], l2 = pl.l2[p], l3 = pl.l3[p];
                int d2 = 2 * l2 + 1, d3 = 2 * l3 + 1;
                const double *Cp = pl.cg[p];
                const double *wp = w + (e * P + p) * C;
                for (int m1 = 0; m1 <= 2 * l1; ++m1)
                    for (int m2 = 0; m2 <= 2 * l2; ++m2)
                        for (int m3 = 0; m3 <= 2 * l3; ++m3) {
                            double c = Cp[(m1 * d2 + m2) * d3 + m3];
                            if (c == 0.0) continue;
                            double cy = c * Ye[l2 * l2 + m2];
                            const double *gb = gr + (pl.out_off[p] + m3) * C;
                            double *db = d + (pl.in_off[p] + m1) * C;
                            for (int u = 0; u < C; ++u) db[u] += wp[u] * cy * gb[u];
                        }
            }
        }
    }
    free(ptr); free(list);
    plan_free(&pl);
    return 0;
}

/* ------------------------------------------------------------------------------------
 * Edge -> atom force reduction (reading A10: r_e = pos[rcv] - pos[snd] + shift):
 *   F_i = -( sum_{e: rcv(e)=i} dvec_e  -  sum_{e: snd(e)=i} dvec_e )
 * ---------------------------------------------------------------------------------- */
void orc_force_reduce(const double *dvec, const int32_t *senders, const int32_t *receivers,
                      int64_t E, int32_t N, double *F)
{
    for (int64_t i = 0; i < (int64_t)N * 3; ++i) F[i] = 0.0;
    for (int64_t e = 0; e < E; ++e)
        for (int a = 0; a < 3; ++a) {
            F[(int64_t)receivers[e] * 3 + a] -= dvec[3 * e + a];
            F[(int64_t)senders[e] * 3 + a] += dvec[3 * e + a];
        }
}
