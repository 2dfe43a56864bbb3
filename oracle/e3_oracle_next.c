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
