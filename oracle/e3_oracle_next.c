/*
 * e3_oracle_next.c -- fp64 CPU ORACLE for the SURVEY.md section 8(f) "NEXT" rows.  TEST INFRASTRUCTURE ONLY.
 *
 * Same rules as e3_oracle.c: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
 * call this; it shares no code, header, table or constant with the CUDA path; plain loops in double precision, written in
 * the order of the definitions quoted below so that a reader can check them by eye.
 *
 * NEXT-1, the radial network that GENERATES the per-edge weights ("fusion of the message passing kernel" is the
 * authors' open item; the paper only names the ingredients: L487 `num_rbf 8`, L488 `radial_net_nonlinearity swish`, L489
 * `radial_net_n_hidden 64`, L490 `radial_net_n_layers 2`, L491 / L542 `radial_envelope polynomial_envelope`, L539 `num_rbf 16`,
 * L497 / L549 `graph_cutoff_angstrom 5.0`).  It prints no formula, so the formulas are readings (R1-R4):
 *   R1  Bessel basis        b_k(r) = sqrt(2/rc) sin(k pi r / rc) / r,  k = 1..K   (limit k pi / rc * sqrt(2/rc) at r = 0)
 *   R2  polynomial envelope u(x) = 1 - (p+1)(p+2)/2 x^p + p(p+2) x^(p+1) - p(p+1)/2 x^(p+2) for x = r/rc < 1, 0 otherwise
 *       (p = 6 unless stated); radial features f_k(r) = b_k(r) u(r/rc)
 *   R3  network             h1 = silu(f W1), h2 = silu(h1 W2), w = h2 W3  with silu(a) = a / (1 + exp(-a)) (= "swish"),
 *       W1[K,H], W2[H,H], W3[H,P*C], no biases ("n_hidden" H = 64, "n_layers" = the two hidden layers)
 *   R4  the weights feed the tensor product unchanged: w[e, p*C + u]; the extra force term is dE/dr * vec/|vec|
 * Pins (tests/test_oracle_radial.py): envelope closed forms u(0) = 1, u(1) = u'(1) = u''(1) = 0 and the p = 6 polynomial typed
 * out; Bessel against a library spherical Bessel j0, its zero at rc and its orthonormality under int r^2 dr; d f / d r against
 * central differences; the network against a vectorised numpy / scipy.special.expit restatement and a hand-typed scalar case;
 * its VJP against central differences of every input and the adjoint identity; forces of the whole path (SH + radial term)
 * against finite differences of the positions, sum F = 0, zero torque.
 *
 * NEXT-2, second-order VJP of the tensor product (section 5.2, Eq. 3-4: Hessian rows are VJPs of the force
 * function): orc_tp_scatter_vjp_vjp below.  NEXT-3, MACE's symmetric contraction at correlation 2 (L535 `node_symmetry 2`, L536
 * `correlation 2`, L545 `symmetric_contraction_backend e3j`): orc_symcon2_*.  NEXT-4, unequal multiplicities: orc_tp_mul_*.
 * Their definitions and pins are stated at each function.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ---------------------------------------------------------------------------------------------------------------
 * R2: polynomial envelope and its derivative with respect to x.
 * ------------------------------------------------------------------------------------------------------------- */
void orc_poly_envelope(int p, int64_t n, const double *x, double *u, double *du)
{
    const double a = -0.5 * (p + 1) * (p + 2), b = (double)p * (p + 2), c = -0.5 * p * (p + 1);
    for (int64_t i = 0; i < n; ++i) {
        const double t = x[i];
        if (t < 1.0) {
            u[i] = 1.0 + a * pow(t, p) + b * pow(t, p + 1) + c * pow(t, p + 2);
            du[i] = a * p * pow(t, p - 1) + b * (p + 1) * pow(t, p) + c * (p + 2) * pow(t, p + 1);
        } else {
            u[i] = 0.0;
            du[i] = 0.0;
        }
    }
}

/* ---------------------------------------------------------------------------------------------------------------
 * R1 + R2: radial features f[i,k] = b_{k+1}(r_i) u(r_i / rc) and d f / d r, k = 0..K-1.
 * ------------------------------------------------------------------------------------------------------------- */
void orc_radial_basis(int K, int p, double rc, int64_t n, const double *r, double *f, double *dfdr)
{
    const double pi = 3.14159265358979323846, nrm = sqrt(2.0 / rc);
    for (int64_t i = 0; i < n; ++i) {
        const double ri = r[i];
        double x = ri / rc, u, du;
        orc_poly_envelope(p, 1, &x, &u, &du);
        for (int k = 0; k < K; ++k) {
            const double a = (k + 1) * pi / rc;
            double b, db;
            if (ri > 0.0) {
                b = nrm * sin(a * ri) / ri;
                db = nrm * (a * cos(a * ri) / ri - sin(a * ri) / (ri * ri));
            } else {
                b = nrm * a;          /* sin(a r) / r -> a */
                db = 0.0;             /* even function of r */
            }
            f[i * K + k] = b * u;
            dfdr[i * K + k] = db * u + b * du / rc;
        }
    }
}

static double silu(double a) { return a / (1.0 + exp(-a)); }
static double dsilu(double a) { const double s = 1.0 / (1.0 + exp(-a)); return s + a * s * (1.0 - s); }

/* ---------------------------------------------------------------------------------------------------------------
 * R3: w[i, :] = silu(silu(f[i,:] W1) W2) W3.   f[n,K], W1[K,H], W2[H,H], W3[H,M], w[n,M]
 * ------------------------------------------------------------------------------------------------------------- */
void orc_radial_mlp_fwd(int K, int H, int M, int64_t n, const double *f, const double *W1, const double *W2, const double *W3, double *w)
{
    double *h1 = (double *)malloc(sizeof(double) * H), *h2 = (double *)malloc(sizeof(double) * H);
    for (int64_t i = 0; i < n; ++i) {
        for (int j = 0; j < H; ++j) {
            double a = 0.0;
            for (int k = 0; k < K; ++k) a += f[i * K + k] * W1[k * H + j];
            h1[j] = silu(a);
        }
        for (int j = 0; j < H; ++j) {
            double a = 0.0;
            for (int q = 0; q < H; ++q) a += h1[q] * W2[q * H + j];
            h2[j] = silu(a);
        }
        for (int m = 0; m < M; ++m) {
            double a = 0.0;
            for (int j = 0; j < H; ++j) a += h2[j] * W3[j * M + m];
            w[i * M + m] = a;
        }
    }
    free(h1); free(h2);
}

/* VJP of R3: given dw[n,M] = dL/dw, returns df[n,K] and the parameter gradients dW1[K,H], dW2[H,H], dW3[H,M] (summed over i
 * in ascending order). */
void orc_radial_mlp_bwd(int K, int H, int M, int64_t n, const double *f, const double *W1, const double *W2, const double *W3,
                        const double *dw, double *df, double *dW1, double *dW2, double *dW3)
{
    double *a1 = (double *)malloc(sizeof(double) * H), *h1 = (double *)malloc(sizeof(double) * H);
    double *a2 = (double *)malloc(sizeof(double) * H), *h2 = (double *)malloc(sizeof(double) * H);
    double *g2 = (double *)malloc(sizeof(double) * H), *g1 = (double *)malloc(sizeof(double) * H);
    memset(dW1, 0, sizeof(double) * K * H); memset(dW2, 0, sizeof(double) * H * H); memset(dW3, 0, sizeof(double) * (size_t)H * M);
    for (int64_t i = 0; i < n; ++i) {
        for (int j = 0; j < H; ++j) { double a = 0.0; for (int k = 0; k < K; ++k) a += f[i * K + k] * W1[k * H + j]; a1[j] = a; h1[j] = silu(a); }
        for (int j = 0; j < H; ++j) { double a = 0.0; for (int q = 0; q < H; ++q) a += h1[q] * W2[q * H + j]; a2[j] = a; h2[j] = silu(a); }
        for (int j = 0; j < H; ++j) {                     /* dL/da2 */
            double s = 0.0;
            for (int m = 0; m < M; ++m) { s += dw[i * M + m] * W3[j * M + m]; dW3[(size_t)j * M + m] += h2[j] * dw[i * M + m]; }
            g2[j] = s * dsilu(a2[j]);
        }
        for (int q = 0; q < H; ++q) {                     /* dL/da1 */
            double s = 0.0;
            for (int j = 0; j < H; ++j) { s += g2[j] * W2[q * H + j]; dW2[q * H + j] += h1[q] * g2[j]; }
            g1[q] = s * dsilu(a1[q]);
        }
        for (int k = 0; k < K; ++k) {
            double s = 0.0;
            for (int j = 0; j < H; ++j) { s += g1[j] * W1[k * H + j]; dW1[k * H + j] += f[i * K + k] * g1[j]; }
            df[i * K + k] = s;
        }
    }
    free(a1); free(h1); free(a2); free(h2); free(g2); free(g1);
}

/* =================================================================================================================
 * General-multiplicity plan used by the NEXT-2 / NEXT-4 functions below.  Reading A7 generalised (NEXT-4, PAPER.md L484-L485:
 * NequIP `target_irreps 64x0e + 64x0o + 32x1o + 32x1e + 32x2e + 32x2o`): every irrep i has its own multiplicity mul_i; a node row is
 * the concatenation of blocks of (2l_i+1)*mul_i elements, index m*mul_i + u inside a block; a path ("uvu") needs
 * mul(i_in) == mul(i_out) and owns mul weights per edge, stored path after path: w[e, w_off(p) + u].
 * ================================================================================================================= */
typedef struct { int l; int parity; int mul; } nx_irrep;
typedef struct { int i_in; int l_sh; int i_out; } nx_path;
double orc_cg_real(int l1, int l2, int l3, double *C);      /* e3_oracle.c (reading A4) */

typedef struct {
    int n_paths, in_size, out_size, sh_dim, w_size;
    int l1[256], l2[256], l3[256], mul[256], in_off[256], out_off[256], w_off[256];
    double *cg[256];
} nplan;

static void nplan_free(nplan *pl) { for (int p = 0; p < pl->n_paths; ++p) free(pl->cg[p]); }

static int nplan_build(nplan *pl, const nx_irrep *ii, int n_in, int sh_lmax, const nx_irrep *io, int n_out, const nx_path *paths, int n_paths)
{
    int in_off[256], out_off[256];
    pl->n_paths = 0;
    if (n_paths > 256 || n_in > 256 || n_out > 256 || n_in < 1 || n_out < 1) return 1;
    pl->in_size = 0;
    for (int i = 0; i < n_in; ++i) { in_off[i] = pl->in_size; pl->in_size += (2 * ii[i].l + 1) * ii[i].mul; }
    pl->out_size = 0;
    for (int i = 0; i < n_out; ++i) { out_off[i] = pl->out_size; pl->out_size += (2 * io[i].l + 1) * io[i].mul; }
    pl->sh_dim = (sh_lmax + 1) * (sh_lmax + 1);
    pl->w_size = 0;
    for (int p = 0; p < n_paths; ++p) pl->cg[p] = NULL;
    pl->n_paths = n_paths;
    for (int p = 0; p < n_paths; ++p) {
        nx_path q = paths[p];
        if (q.i_in < 0 || q.i_in >= n_in || q.i_out < 0 || q.i_out >= n_out || q.l_sh < 0 || q.l_sh > sh_lmax) return 3;
        const int l1 = ii[q.i_in].l, l2 = q.l_sh, l3 = io[q.i_out].l;
        if (l3 < abs(l1 - l2) || l3 > l1 + l2) return 4;
        if (ii[q.i_in].parity * ((l2 & 1) ? -1 : 1) != io[q.i_out].parity) return 5;
        if (ii[q.i_in].mul != io[q.i_out].mul || ii[q.i_in].mul < 1) return 2;
        pl->l1[p] = l1; pl->l2[p] = l2; pl->l3[p] = l3; pl->mul[p] = ii[q.i_in].mul;
        pl->in_off[p] = in_off[q.i_in]; pl->out_off[p] = out_off[q.i_out];
        pl->w_off[p] = pl->w_size; pl->w_size += pl->mul[p];
        pl->cg[p] = (double *)malloc(sizeof(double) * (size_t)((2 * l1 + 1) * (2 * l2 + 1) * (2 * l3 + 1)));
        orc_cg_real(l1, l2, l3, pl->cg[p]);
    }
    return 0;
}

int orc_tp_mul_dims(const nx_irrep *ii, int n_in, int sh_lmax, const nx_irrep *io, int n_out, const nx_path *paths, int n_paths,
                    int *in_size, int *sh_dim, int *out_size, int *w_size)
{
    nplan pl;
    int rc = nplan_build(&pl, ii, n_in, sh_lmax, io, n_out, paths, n_paths);
    if (!rc) { *in_size = pl.in_size; *sh_dim = pl.sh_dim; *out_size = pl.out_size; *w_size = pl.w_size; }
    nplan_free(&pl);
    return rc;
}

/* NEXT-4: forward with per-irrep multiplicities (the definition of SURVEY 8(c) with C replaced by mul(p)):
 *   out[r, out_off(p) + m3*mul + u] += w[e, w_off(p)+u] * C^p[m1,m2,m3] * x[snd(e), in_off(p) + m1*mul + u] * Y[e, l2^2 + m2]
 * Pins (tests/test_oracle_next.py): equals orc_tp_scatter_fwd for equal multiplicities; brute-force einsum; a plan whose irreps
 * fall into multiplicity classes equals the independent equal-multiplicity plans of the classes. */
int orc_tp_mul_fwd(const nx_irrep *ii, int n_in, int sh_lmax, const nx_irrep *io, int n_out, const nx_path *paths, int n_paths,
                   const double *x, const double *sh, const double *w, const int32_t *senders, const int32_t *receivers, int64_t E, int32_t N, double *out)
{
    nplan pl;
    int rc = nplan_build(&pl, ii, n_in, sh_lmax, io, n_out, paths, n_paths);
    if (rc) { nplan_free(&pl); return rc; }
    memset(out, 0, sizeof(double) * (size_t)N * pl.out_size);
    for (int64_t e = 0; e < E; ++e) {
        const double *xs = x + (int64_t)senders[e] * pl.in_size, *Ye = sh + e * pl.sh_dim, *we = w + e * pl.w_size;
        double *o = out + (int64_t)receivers[e] * pl.out_size;
        for (int p = 0; p < pl.n_paths; ++p) {
            const int l1 = pl.l1[p], l2 = pl.l2[p], l3 = pl.l3[p], mu = pl.mul[p], d2 = 2 * l2 + 1, d3 = 2 * l3 + 1;
            for (int m1 = 0; m1 <= 2 * l1; ++m1)
                for (int m2 = 0; m2 <= 2 * l2; ++m2)
                    for (int m3 = 0; m3 <= 2 * l3; ++m3) {
                        const double c = pl.cg[p][(m1 * d2 + m2) * d3 + m3];
                        if (c == 0.0) continue;
                        for (int u = 0; u < mu; ++u)
                            o[pl.out_off[p] + m3 * mu + u] += we[pl.w_off[p] + u] * c * xs[pl.in_off[p] + m1 * mu + u] * Ye[l2 * l2 + m2];
                    }
        }
    }
    nplan_free(&pl);
    return 0;
}

/* NEXT-4: the three VJP contractions of SURVEY 8(a) a5 with per-irrep multiplicities. */
int orc_tp_mul_bwd(const nx_irrep *ii, int n_in, int sh_lmax, const nx_irrep *io, int n_out, const nx_path *paths, int n_paths,
                   const double *x, const double *sh, const double *w, const int32_t *senders, const int32_t *receivers, int64_t E, int32_t N,
                   const double *g, double *dx, double *dY, double *dw)
{
    nplan pl;
    int rc = nplan_build(&pl, ii, n_in, sh_lmax, io, n_out, paths, n_paths);
    if (rc) { nplan_free(&pl); return rc; }
    memset(dx, 0, sizeof(double) * (size_t)N * pl.in_size);
    memset(dY, 0, sizeof(double) * (size_t)E * pl.sh_dim);
    memset(dw, 0, sizeof(double) * (size_t)E * pl.w_size);
    for (int64_t e = 0; e < E; ++e) {
        const int64_t s = senders[e], r = receivers[e];
        for (int p = 0; p < pl.n_paths; ++p) {
            const int l1 = pl.l1[p], l2 = pl.l2[p], l3 = pl.l3[p], mu = pl.mul[p], d2 = 2 * l2 + 1, d3 = 2 * l3 + 1;
            for (int m1 = 0; m1 <= 2 * l1; ++m1)
                for (int m2 = 0; m2 <= 2 * l2; ++m2)
                    for (int m3 = 0; m3 <= 2 * l3; ++m3) {
                        const double c = pl.cg[p][(m1 * d2 + m2) * d3 + m3];
                        if (c == 0.0) continue;
                        for (int u = 0; u < mu; ++u) {
                            const double xv = x[s * pl.in_size + pl.in_off[p] + m1 * mu + u], Yv = sh[e * pl.sh_dim + l2 * l2 + m2];
                            const double wv = w[e * pl.w_size + pl.w_off[p] + u], gv = g[r * pl.out_size + pl.out_off[p] + m3 * mu + u];
                            dx[s * pl.in_size + pl.in_off[p] + m1 * mu + u] += c * Yv * wv * gv;
                            dY[e * pl.sh_dim + l2 * l2 + m2] += c * xv * wv * gv;
                            dw[e * pl.w_size + pl.w_off[p] + u] += c * xv * Yv * gv;
                        }
                    }
        }
    }
    nplan_free(&pl);
    return 0;
}

/* NEXT-2: VJP of the VJP (section 5.2, Eq. 3-4: a Hessian row is a reverse-mode derivative of selected force
 * components, i.e. of first-order VJP outputs).  The forward is trilinear, T = sum C x Y w, and the first-order outputs for a cotangent g
 * are dx = sum C Y w g, dY = sum C x w g, dw = sum C x Y g.  For cotangents (vx, vY, vw) of (dx, dY, dw) the scalar
 *   S = <vx, dx> + <vY, dY> + <vw, dw> = sum C g (vx Y w + x vY w + x Y vw)
 * has the gradients written out below (each is S with one factor removed):
 *   gg = dS/dg, gx = dS/dx, gY = dS/dY, gw = dS/dw.
 * Pins: central differences of S built from the (pinned) first-order oracle in every input; gg = T(vx,Y,w) + T(x,vY,w) + T(x,Y,vw)
 * through orc_tp_scatter_fwd; symmetry of the second derivative. */
int orc_tp_vjp_vjp(const nx_irrep *ii, int n_in, int sh_lmax, const nx_irrep *io, int n_out, const nx_path *paths, int n_paths,
                   const double *x, const double *sh, const double *w, const int32_t *senders, const int32_t *receivers, int64_t E, int32_t N,
                   const double *g, const double *vx, const double *vY, const double *vw,
                   double *gg, double *gx, double *gY, double *gw)
{
    nplan pl;
    int rc = nplan_build(&pl, ii, n_in, sh_lmax, io, n_out, paths, n_paths);
    if (rc) { nplan_free(&pl); return rc; }
    memset(gg, 0, sizeof(double) * (size_t)N * pl.out_size);
    memset(gx, 0, sizeof(double) * (size_t)N * pl.in_size);
    memset(gY, 0, sizeof(double) * (size_t)E * pl.sh_dim);
    memset(gw, 0, sizeof(double) * (size_t)E * pl.w_size);
    for (int64_t e = 0; e < E; ++e) {
        const int64_t s = senders[e], r = receivers[e];
        for (int p = 0; p < pl.n_paths; ++p) {
            const int l1 = pl.l1[p], l2 = pl.l2[p], l3 = pl.l3[p], mu = pl.mul[p], d2 = 2 * l2 + 1, d3 = 2 * l3 + 1;
            for (int m1 = 0; m1 <= 2 * l1; ++m1)
                for (int m2 = 0; m2 <= 2 * l2; ++m2)
                    for (int m3 = 0; m3 <= 2 * l3; ++m3) {
                        const double c = pl.cg[p][(m1 * d2 + m2) * d3 + m3];
                        if (c == 0.0) continue;
                        for (int u = 0; u < mu; ++u) {
                            const int64_t ix = s * pl.in_size + pl.in_off[p] + m1 * mu + u, iy = e * pl.sh_dim + l2 * l2 + m2;
                            const int64_t iw = e * pl.w_size + pl.w_off[p] + u, ig = r * pl.out_size + pl.out_off[p] + m3 * mu + u;
                            const double xv = x[ix], Yv = sh[iy], wv = w[iw], gv = g[ig], a = vx[ix], b = vY[iy], d = vw[iw];
                            gg[ig] += c * (a * Yv * wv + xv * b * wv + xv * Yv * d);
                            gx[ix] += c * gv * (b * wv + Yv * d);
                            gY[iy] += c * gv * (a * wv + xv * d);
                            gw[iw] += c * gv * (a * Yv + xv * b);
                        }
                    }
        }
    }
    nplan_free(&pl);
    return 0;
}

/* NEXT-2: second derivative of the spherical harmonics, as the VJP of  (vec, dY) -> dvec = J(vec)^T dY  (orc_sh_bwd) for a
 * cotangent u[n,3]:   g_dY[n,lm] = J(vec) u   and   g_vec = (sum_lm dY_lm Hess Y_lm(vec)) u.
 * Y_lm(vec) = P_lm(vec) / |vec|^l with the homogeneous polynomials P_lm of reading A2 (the explicit forms with 1 written as r^2), kept
 * here as monomial tables; gradient and Hessian follow from
 *   grad f = grad P r^-l - l P r^-(l+2) v,
 *   Hess f = Hess P r^-l - l (grad P v^T + v grad P^T) r^-(l+2) - l P r^-(l+2) I + l (l+2) P r^-(l+4) v v^T.
 * A zero vector gives zeros (reading A3).  Pins: P/r^l equals orc_sh; g_dY equals orc_sh_jac applied to u; g_vec equals central
 * differences of orc_sh_bwd; Hess is symmetric and annihilates ... r (degree-0 homogeneity: Hess f v = -grad f). */
typedef struct { double c; int a, b, d; } mono;   /* c x^a y^b z^d */
#define S3 1.7320508075688772935
#define S5 2.2360679774997896964
#define S7 2.6457513110645905905
#define S15 3.8729833462074168852
#define S42 6.4807406984078602310
#define S70 8.3666002653407554798
#define S105 10.246950765959598383
static const mono P00[] = { { 1.0, 0, 0, 0 } };
static const mono P1m[] = { { S3, 0, 1, 0 } }, P10[] = { { S3, 0, 0, 1 } }, P1p[] = { { S3, 1, 0, 0 } };
static const mono P2a[] = { { S15, 1, 1, 0 } }, P2b[] = { { S15, 0, 1, 1 } };
static const mono P2c[] = { { S5, 0, 0, 2 }, { -0.5 * S5, 2, 0, 0 }, { -0.5 * S5, 0, 2, 0 } };          /* (sqrt5/2)(3z^2 - r^2) */
static const mono P2d[] = { { S15, 1, 0, 1 } }, P2e[] = { { 0.5 * S15, 2, 0, 0 }, { -0.5 * S15, 0, 2, 0 } };
static const mono P3a[] = { { 0.75 * S70, 2, 1, 0 }, { -0.25 * S70, 0, 3, 0 } };                          /* (sqrt70/4) y (3x^2 - y^2) */
static const mono P3b[] = { { S105, 1, 1, 1 } };
static const mono P3c[] = { { S42, 0, 1, 2 }, { -0.25 * S42, 2, 1, 0 }, { -0.25 * S42, 0, 3, 0 } };      /* (sqrt42/4) y (5z^2 - r^2) */
static const mono P3d[] = { { S7, 0, 0, 3 }, { -1.5 * S7, 2, 0, 1 }, { -1.5 * S7, 0, 2, 1 } };           /* (sqrt7/2) z (5z^2 - 3r^2) */
static const mono P3e[] = { { S42, 1, 0, 2 }, { -0.25 * S42, 3, 0, 0 }, { -0.25 * S42, 1, 2, 0 } };      /* (sqrt42/4) x (5z^2 - r^2) */
static const mono P3f[] = { { 0.5 * S105, 2, 0, 1 }, { -0.5 * S105, 0, 2, 1 } };
static const mono P3g[] = { { 0.25 * S70, 3, 0, 0 }, { -0.75 * S70, 1, 2, 0 } };                          /* (sqrt70/4) x (x^2 - 3y^2) */
static const mono *const PT[16] = { P00, P1m, P10, P1p, P2a, P2b, P2c, P2d, P2e, P3a, P3b, P3c, P3d, P3e, P3f, P3g };
static const int PN[16] = { 1, 1, 1, 1, 1, 1, 3, 1, 2, 2, 1, 3, 3, 3, 2, 2 };
static const int PL[16] = { 0, 1, 1, 1, 2, 2, 2, 2, 2, 3, 3, 3, 3, 3, 3, 3 };

static double ipow(double t, int n) { double r = 1.0; for (int i = 0; i < n; ++i) r *= t; return r; }

/* value, gradient and Hessian of the polynomial P_lm at v */
static void poly_eval(int lm, const double *v, double *P, double *gP, double *HP)
{
    *P = 0.0;
    for (int i = 0; i < 3; ++i) gP[i] = 0.0;
    for (int i = 0; i < 9; ++i) HP[i] = 0.0;
    for (int t = 0; t < PN[lm]; ++t) {
        const mono m = PT[lm][t];
        const int ex[3] = { m.a, m.b, m.d };
        *P += m.c * ipow(v[0], ex[0]) * ipow(v[1], ex[1]) * ipow(v[2], ex[2]);
        for (int i = 0; i < 3; ++i) {
            if (ex[i] < 1) continue;
            int e1[3] = { ex[0], ex[1], ex[2] };
            e1[i] -= 1;
            const double ci = m.c * ex[i];
            gP[i] += ci * ipow(v[0], e1[0]) * ipow(v[1], e1[1]) * ipow(v[2], e1[2]);
            for (int j = 0; j < 3; ++j) {
                if (e1[j] < 1) continue;
                int e2[3] = { e1[0], e1[1], e1[2] };
                e2[j] -= 1;
                HP[i * 3 + j] += ci * e1[j] * ipow(v[0], e2[0]) * ipow(v[1], e2[1]) * ipow(v[2], e2[2]);
            }
        }
    }
}

int orc_sh_bwd_bwd(int lmax, int64_t n, const double *vec, const double *dY, const double *u, double *g_vec, double *g_dY)
{
    if (lmax < 0 || lmax > 3) return 1;
    const int D = (lmax + 1) * (lmax + 1);
    for (int64_t i = 0; i < n; ++i) {
        const double *v = vec + 3 * i, *ui = u + 3 * i;
        double *gv = g_vec + 3 * i;
        gv[0] = gv[1] = gv[2] = 0.0;
        const double r2 = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
        if (!(r2 > 0.0)) { for (int k = 0; k < D; ++k) g_dY[i * D + k] = 0.0; continue; }
        const double r = sqrt(r2);
        for (int lm = 0; lm < D; ++lm) {
            const int l = PL[lm];
            double P, gP[3], HP[9];
            poly_eval(lm, v, &P, gP, HP);
            const double rl = ipow(r, l);
            double grad[3], H[9];
            for (int a = 0; a < 3; ++a) grad[a] = gP[a] / rl - l * P / (rl * r2) * v[a];
            for (int a = 0; a < 3; ++a)
                for (int b = 0; b < 3; ++b)
                    H[a * 3 + b] = HP[a * 3 + b] / rl - l * (gP[a] * v[b] + v[a] * gP[b]) / (rl * r2) - (a == b ? l * P / (rl * r2) : 0.0)
                                   + l * (l + 2) * P / (rl * r2 * r2) * v[a] * v[b];
            g_dY[i * D + lm] = grad[0] * ui[0] + grad[1] * ui[1] + grad[2] * ui[2];
            for (int a = 0; a < 3; ++a) gv[a] += dY[i * D + lm] * (H[a * 3] * ui[0] + H[a * 3 + 1] * ui[1] + H[a * 3 + 2] * ui[2]);
        }
    }
    return 0;
}

/* =================================================================================================================
 * NEXT-3: MACE's symmetric contraction at correlation order 2 on node features (PAPER.md L535 `node_symmetry 2`, L536
 * `correlation 2`, L545 `symmetric_contraction_backend e3j`; the paper prints no formula).  Reading S1: for node n of
 * species z_n, channel u, every path carries one weight per species and channel, W[z, path, u]; a path is either
 *   linear     (i_in1, -1,    i_out):  B[n, i_out, M, u] += W * A[n, i_in1, M, u]                      (correlation 1; same l and parity)
 *   quadratic  (i_in1, i_in2, i_out):  B[n, i_out, M, u] += W * sum_{m1,m2} C^{l1 l2 L}[m1,m2,M] A[n,i_in1,m1,u] A[n,i_in2,m2,u]
 * with the real CG tensors of reading A4 (triangle rule, parity p1*p2 = p_out).  Layout as everywhere (A7): block after block,
 * index m*C + u.  All irreps share one multiplicity C.
 * Pins (tests/test_oracle_next.py): brute-force einsum; Wigner-D equivariance and inversion; L = 0 closed form
 * (-1)^l/sqrt(2l+1) |A_l|^2; the antisymmetric 1x1->1 self-product vanishes; VJP vs central differences and Euler's identity
 * (the map is linear + quadratic in A).
 * ================================================================================================================= */
typedef struct { int i_in1; int i_in2; int i_out; } sc_path;

static int sc_offsets(const nx_irrep *ir, int n, int *off) { int o = 0; for (int i = 0; i < n; ++i) { off[i] = o; o += 2 * ir[i].l + 1; } return o; }

static int sc_check(const nx_irrep *ii, int n_in, const nx_irrep *io, int n_out, const sc_path *paths, int n_paths)
{
    if (n_in < 1 || n_out < 1 || n_paths < 1 || n_in > 64 || n_out > 64) return 1;
    const int C = ii[0].mul;
    for (int i = 0; i < n_in; ++i) if (ii[i].mul != C) return 2;
    for (int i = 0; i < n_out; ++i) if (io[i].mul != C) return 2;
    for (int p = 0; p < n_paths; ++p) {
        const sc_path q = paths[p];
        if (q.i_in1 < 0 || q.i_in1 >= n_in || q.i_in2 >= n_in || q.i_out < 0 || q.i_out >= n_out) return 3;
        if (q.i_in2 < 0) {
            if (ii[q.i_in1].l != io[q.i_out].l || ii[q.i_in1].parity != io[q.i_out].parity) return 4;
        } else {
            const int l1 = ii[q.i_in1].l, l2 = ii[q.i_in2].l, L = io[q.i_out].l;
            if (L < abs(l1 - l2) || L > l1 + l2) return 4;
            if (ii[q.i_in1].parity * ii[q.i_in2].parity != io[q.i_out].parity) return 5;
        }
    }
    return 0;
}

int orc_symcon2_fwd(const nx_irrep *ii, int n_in, const nx_irrep *io, int n_out, const sc_path *paths, int n_paths, int n_species,
                    const double *A, const int32_t *species, const double *W, int32_t N, double *B)
{
    int rc = sc_check(ii, n_in, io, n_out, paths, n_paths);
    if (rc) return rc;
    int in_off[64], out_off[64];
    const int in_dim = sc_offsets(ii, n_in, in_off), out_dim = sc_offsets(io, n_out, out_off), C = ii[0].mul;
    memset(B, 0, sizeof(double) * (size_t)N * out_dim * C);
    for (int p = 0; p < n_paths; ++p) {
        const sc_path q = paths[p];
        const int L = io[q.i_out].l;
        double *cg = NULL;
        int l1 = ii[q.i_in1].l, l2 = 0;
        if (q.i_in2 >= 0) { l2 = ii[q.i_in2].l; cg = (double *)malloc(sizeof(double) * (size_t)((2 * l1 + 1) * (2 * l2 + 1) * (2 * L + 1))); orc_cg_real(l1, l2, L, cg); }
        for (int32_t n = 0; n < N; ++n) {
            if (species[n] < 0 || species[n] >= n_species) { free(cg); return 6; }
            const double *a = A + (int64_t)n * in_dim * C, *w = W + ((int64_t)species[n] * n_paths + p) * C;
            double *b = B + (int64_t)n * out_dim * C;
            for (int u = 0; u < C; ++u) {
                if (q.i_in2 < 0) {
                    for (int M = 0; M <= 2 * L; ++M) b[(out_off[q.i_out] + M) * C + u] += w[u] * a[(in_off[q.i_in1] + M) * C + u];
                } else {
                    for (int m1 = 0; m1 <= 2 * l1; ++m1)
                        for (int m2 = 0; m2 <= 2 * l2; ++m2)
                            for (int M = 0; M <= 2 * L; ++M)
                                b[(out_off[q.i_out] + M) * C + u] += w[u] * cg[(m1 * (2 * l2 + 1) + m2) * (2 * L + 1) + M] *
                                                                     a[(in_off[q.i_in1] + m1) * C + u] * a[(in_off[q.i_in2] + m2) * C + u];
                }
            }
        }
        free(cg);
    }
    return 0;
}

/* VJP: dA[N,in_dim*C] and dW[S,n_paths,C] (summed over the nodes of each species in ascending node order) for a cotangent g = dL/dB */
int orc_symcon2_bwd(const nx_irrep *ii, int n_in, const nx_irrep *io, int n_out, const sc_path *paths, int n_paths, int n_species,
                    const double *A, const int32_t *species, const double *W, int32_t N, const double *g, double *dA, double *dW)
{
    int rc = sc_check(ii, n_in, io, n_out, paths, n_paths);
    if (rc) return rc;
    int in_off[64], out_off[64];
    const int in_dim = sc_offsets(ii, n_in, in_off), out_dim = sc_offsets(io, n_out, out_off), C = ii[0].mul;
    memset(dA, 0, sizeof(double) * (size_t)N * in_dim * C);
    memset(dW, 0, sizeof(double) * (size_t)n_species * n_paths * C);
    for (int p = 0; p < n_paths; ++p) {
        const sc_path q = paths[p];
        const int L = io[q.i_out].l;
        double *cg = NULL;
        int l1 = ii[q.i_in1].l, l2 = 0;
        if (q.i_in2 >= 0) { l2 = ii[q.i_in2].l; cg = (double *)malloc(sizeof(double) * (size_t)((2 * l1 + 1) * (2 * l2 + 1) * (2 * L + 1))); orc_cg_real(l1, l2, L, cg); }
        for (int32_t n = 0; n < N; ++n) {
            if (species[n] < 0 || species[n] >= n_species) { free(cg); return 6; }
            const double *a = A + (int64_t)n * in_dim * C, *w = W + ((int64_t)species[n] * n_paths + p) * C, *gn = g + (int64_t)n * out_dim * C;
            double *da = dA + (int64_t)n * in_dim * C, *dw = dW + ((int64_t)species[n] * n_paths + p) * C;
            for (int u = 0; u < C; ++u) {
                if (q.i_in2 < 0) {
                    for (int M = 0; M <= 2 * L; ++M) {
                        const double gv = gn[(out_off[q.i_out] + M) * C + u];
                        da[(in_off[q.i_in1] + M) * C + u] += w[u] * gv;
                        dw[u] += a[(in_off[q.i_in1] + M) * C + u] * gv;
                    }
                } else {
                    for (int m1 = 0; m1 <= 2 * l1; ++m1)
                        for (int m2 = 0; m2 <= 2 * l2; ++m2)
                            for (int M = 0; M <= 2 * L; ++M) {
                                const double c = cg[(m1 * (2 * l2 + 1) + m2) * (2 * L + 1) + M], gv = gn[(out_off[q.i_out] + M) * C + u];
                                const double a1 = a[(in_off[q.i_in1] + m1) * C + u], a2 = a[(in_off[q.i_in2] + m2) * C + u];
                                da[(in_off[q.i_in1] + m1) * C + u] += w[u] * c * a2 * gv;
                                da[(in_off[q.i_in2] + m2) * C + u] += w[u] * c * a1 * gv;
                                dw[u] += c * a1 * a2 * gv;
                            }
                }
            }
        }
        free(cg);
    }
    return 0;
}
