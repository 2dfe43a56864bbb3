// Plan construction: path-table validation, the Clebsch-Gordan planner kernel
// (fp64 on the device, Racah closed form + real-basis change, reading A4), sparse tables and the
// partition of the output irreps into forward "roles".
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <functional>
#include <map>
#include <string>

#include "e3_internal.h"

namespace e3 {

// ---------------------------------------------------------------------------------------------
// thread-local error text
// ---------------------------------------------------------------------------------------------
static thread_local char g_err[16384] = "";

void set_error(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}
const char *get_error() { return g_err; }
int cuda_fail(cudaError_t e, const char *what)
{
    set_error("CUDA error %d (%s) in %s", (int)e, cudaGetErrorString(e), what);
    cudaGetLastError();   // clear sticky-less errors
    return E3_ERR_CUDA;
}

// ---------------------------------------------------------------------------------------------
// Clebsch-Gordan coefficients.  One routine, compiled for host and device; the plan uses the
// device instantiation (kernel `cg_planner_kernel`), e3_jit_check the host one.
//
// Complex (Condon-Shortley) coefficient, Racah's closed form (reading A4):
//   <l1 a l2 b | l3 c> = [c == a+b] sqrt( (2l3+1) (l3+l1-l2)! (l3-l1+l2)! (l1+l2-l3)! / (l1+l2+l3+1)! )
//        * sqrt( (l3+c)! (l3-c)! (l1-a)! (l1+a)! (l2-b)! (l2+b)! )
//        * sum_k (-1)^k / ( k! (l1+l2-l3-k)! (l1-a-k)! (l2+b-k)! (l3-l2+a+k)! (l3-l1-b+k)! )
// Real tensor: C[m1,m2,m3] = Re or Im (even / odd l1+l2+l3) of
//   sum_{mu1,mu2} U1[m1,mu1] U2[m2,mu2] conj(U3[m3,mu1+mu2]) <l1 mu1 l2 mu2 | l3 mu1+mu2>
// with U the complex->real change of basis of reading A1.  A row of U has at most two entries
// (mu = -|m| and mu = +|m|), so the sum has at most four terms.
// ---------------------------------------------------------------------------------------------
struct Cx { double re, im; };
__host__ __device__ inline Cx cx_mul(Cx a, Cx b) { return { a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re }; }

__host__ __device__ inline double factorial_d(int n)
{
    const double t[14] = { 1., 1., 2., 6., 24., 120., 720., 5040., 40320., 362880., 3628800., 39916800.,
                           479001600., 6227020800. };
    return t[n];
}

__host__ __device__ inline double cg_complex_racah(int l1, int a, int l2, int b, int l3, int c)
{
    if (a + b != c) return 0.0;
    if (l3 < (l1 > l2 ? l1 - l2 : l2 - l1) || l3 > l1 + l2) return 0.0;
    if (a < -l1 || a > l1 || b < -l2 || b > l2 || c < -l3 || c > l3) return 0.0;
    double tri = (2.0 * l3 + 1.0) * factorial_d(l3 + l1 - l2) * factorial_d(l3 - l1 + l2) * factorial_d(l1 + l2 - l3)
                 / factorial_d(l1 + l2 + l3 + 1);
    double mm = factorial_d(l3 + c) * factorial_d(l3 - c) * factorial_d(l1 - a) * factorial_d(l1 + a)
                * factorial_d(l2 - b) * factorial_d(l2 + b);
    double s = 0.0;
    int kmin = 0;
    if (l2 - l3 - a > kmin) kmin = l2 - l3 - a;
    if (l1 - l3 + b > kmin) kmin = l1 - l3 + b;
    int kmax = l1 + l2 - l3;
    if (l1 - a < kmax) kmax = l1 - a;
    if (l2 + b < kmax) kmax = l2 + b;
    for (int k = kmin; k <= kmax; ++k) {
        double den = factorial_d(k) * factorial_d(l1 + l2 - l3 - k) * factorial_d(l1 - a - k) * factorial_d(l2 + b - k)
                     * factorial_d(l3 - l2 + a + k) * factorial_d(l3 - l1 - b + k);
        s += ((k & 1) ? -1.0 : 1.0) / den;
    }
    return sqrt(tri) * sqrt(mm) * s;
}

// entry U[m, mu] of the complex->real basis change (m, mu are true indices, -l..l)
__host__ __device__ inline Cx basis_U(int m, int mu)
{
    const double h = 0.70710678118654752440;
    int a = m < 0 ? -m : m;
    if (mu != a && mu != -a) return { 0.0, 0.0 };
    if (m == 0) return { 1.0, 0.0 };
    double sg = (a & 1) ? -1.0 : 1.0;
    if (m > 0) return (mu < 0) ? Cx{ h, 0.0 } : Cx{ sg * h, 0.0 };
    return (mu < 0) ? Cx{ 0.0, h } : Cx{ 0.0, -sg * h };
}

// one element of the real CG tensor; m1,m2,m3 are 0-based (m_true + l)
__host__ __device__ inline double cg_real_element(int l1, int l2, int l3, int i1, int i2, int i3)
{
    int m1 = i1 - l1, m2 = i2 - l2, m3 = i3 - l3;
    int a1 = m1 < 0 ? -m1 : m1, a2 = m2 < 0 ? -m2 : m2;
    Cx acc = { 0.0, 0.0 };
    for (int s1 = -1; s1 <= 1; s1 += 2) {
        if (a1 == 0 && s1 > 0) continue;
        int mu1 = s1 * a1;
        for (int s2 = -1; s2 <= 1; s2 += 2) {
            if (a2 == 0 && s2 > 0) continue;
            int mu2 = s2 * a2;
            int mu3 = mu1 + mu2;
            if (mu3 < -l3 || mu3 > l3) continue;
            Cx u3 = basis_U(m3, mu3);
            if (u3.re == 0.0 && u3.im == 0.0) continue;
            double c = cg_complex_racah(l1, mu1, l2, mu2, l3, mu3);
            Cx t = cx_mul(cx_mul(basis_U(m1, mu1), basis_U(m2, mu2)), Cx{ u3.re, -u3.im });
            acc.re += t.re * c;
            acc.im += t.im * c;
        }
    }
    return ((l1 + l2 + l3) & 1) ? acc.im : acc.re;
}

double cg_real_host(int l1, int l2, int l3, int m1, int m2, int m3) { return cg_real_element(l1, l2, l3, m1, m2, m3); }

// Planner kernel: one thread per element of every requested dense tensor.
__global__ void cg_planner_kernel(const int *__restrict__ triples, const int *__restrict__ offsets, int n_triples,
                                  int total, double *__restrict__ dense)
{
    int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total) return;
    int t = 0;
    while (t + 1 < n_triples && offsets[t + 1] <= idx) ++t;
    int l1 = triples[3 * t], l2 = triples[3 * t + 1], l3 = triples[3 * t + 2];
    int local = idx - offsets[t];
    int d2 = 2 * l2 + 1, d3 = 2 * l3 + 1;
    int i3 = local % d3, i2 = (local / d3) % d2, i1 = local / (d3 * d2);
    dense[idx] = cg_real_element(l1, l2, l3, i1, i2, i3);
}

int launch_cg_planner(const int *triples, int n, std::vector<std::vector<double>> &dense_out)
{
    std::vector<int> off(n + 1, 0);
    for (int t = 0; t < n; ++t)
        off[t + 1] = off[t] + (2 * triples[3 * t] + 1) * (2 * triples[3 * t + 1] + 1) * (2 * triples[3 * t + 2] + 1);
    int total = off[n];
    int *d_tr = nullptr, *d_off = nullptr;
    double *d_dense = nullptr;
    std::vector<double> flat(total);
    // legacy default stream + blocking copies: e3_plan_create is documented to synchronise
    cudaError_t e = cudaMalloc(&d_tr, sizeof(int) * 3 * n);
    if (e == cudaSuccess) e = cudaMalloc(&d_off, sizeof(int) * (n + 1));
    if (e == cudaSuccess) e = cudaMalloc(&d_dense, sizeof(double) * total);
    if (e == cudaSuccess) e = cudaMemcpy(d_tr, triples, sizeof(int) * 3 * n, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(d_off, off.data(), sizeof(int) * (n + 1), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        cg_planner_kernel<<<(total + 127) / 128, 128>>>(d_tr, d_off, n, total, d_dense);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpy(flat.data(), d_dense, sizeof(double) * total, cudaMemcpyDeviceToHost);
    cudaFree(d_tr); cudaFree(d_off); cudaFree(d_dense);      // on every path
    if (e != cudaSuccess) return cuda_fail(e, "cg planner");
    dense_out.resize(n);
    for (int t = 0; t < n; ++t) dense_out[t].assign(flat.begin() + off[t], flat.begin() + off[t + 1]);
    return E3_OK;
}

// ---------------------------------------------------------------------------------------------
// tables
// ---------------------------------------------------------------------------------------------
int plan_build_tables(e3_plan &pl, const e3_irrep *irreps_in, int n_in, int sh_lmax, const e3_irrep *irreps_out,
                      int n_out, const e3_path *paths, int n_paths, e3_dtype dtype, bool cg_on_device)
{
    if (!irreps_in || !irreps_out || !paths || n_in < 1 || n_out < 1 || n_paths < 1) {
        set_error("plan: null or empty irreps / path table");
        return E3_ERR_INVALID_ARG;
    }
    if (dtype != E3_F32 && dtype != E3_BF16) { set_error("plan: unknown dtype %d", (int)dtype); return E3_ERR_INVALID_ARG; }
    if (sh_lmax < 0 || sh_lmax > kMaxL) { set_error("plan: sh_lmax %d not in 0..%d", sh_lmax, kMaxL); return E3_ERR_UNSUPPORTED; }
    pl.irreps_in.assign(irreps_in, irreps_in + n_in);
    pl.irreps_out.assign(irreps_out, irreps_out + n_out);
    pl.sh_lmax = sh_lmax;
    pl.sh_dim = (sh_lmax + 1) * (sh_lmax + 1);
    pl.dtype = dtype;
    pl.C = irreps_in[0].mul;
    if (pl.C < 1) { set_error("plan: multiplicity must be >= 1"); return E3_ERR_INVALID_ARG; }
    std::vector<int> in_off(n_in), out_off(n_out);
    pl.in_dim = 0;
    for (int i = 0; i < n_in; ++i) {
        const e3_irrep &r = irreps_in[i];
        if (r.l < 0 || (r.parity != 1 && r.parity != -1)) { set_error("plan: bad input irrep %d", i); return E3_ERR_INVALID_ARG; }
        if (r.l > kMaxL) { set_error("plan: input irrep %d has l=%d > %d", i, r.l, kMaxL); return E3_ERR_UNSUPPORTED; }
        if (r.mul != pl.C) { set_error("plan: unequal multiplicities are not supported"); return E3_ERR_UNSUPPORTED; }
        in_off[i] = pl.in_dim;
        pl.in_dim += 2 * r.l + 1;
    }
    pl.out_dim = 0;
    for (int i = 0; i < n_out; ++i) {
        const e3_irrep &r = irreps_out[i];
        if (r.l < 0 || (r.parity != 1 && r.parity != -1)) { set_error("plan: bad output irrep %d", i); return E3_ERR_INVALID_ARG; }
        if (r.l > kMaxL) { set_error("plan: output irrep %d has l=%d > %d", i, r.l, kMaxL); return E3_ERR_UNSUPPORTED; }
        if (r.mul != pl.C) { set_error("plan: unequal multiplicities are not supported"); return E3_ERR_UNSUPPORTED; }
        out_off[i] = pl.out_dim;
        pl.out_dim += 2 * r.l + 1;
    }
    pl.paths.clear();
    std::vector<int> triples;
    for (int p = 0; p < n_paths; ++p) {
        const e3_path &q = paths[p];
        if (q.i_in < 0 || q.i_in >= n_in || q.i_out < 0 || q.i_out >= n_out || q.l_sh < 0 || q.l_sh > sh_lmax) {
            set_error("plan: path %d has an index out of range", p);
            return E3_ERR_BAD_PATH;
        }
        PathInfo pi;
        pi.i_in = q.i_in; pi.l_sh = q.l_sh; pi.i_out = q.i_out;
        pi.l1 = irreps_in[q.i_in].l; pi.l2 = q.l_sh; pi.l3 = irreps_out[q.i_out].l;
        if (pi.l3 < std::abs(pi.l1 - pi.l2) || pi.l3 > pi.l1 + pi.l2) {
            set_error("plan: path %d (%d x %d -> %d) violates the triangle rule", p, pi.l1, pi.l2, pi.l3);
            return E3_ERR_BAD_PATH;
        }
        int par = irreps_in[q.i_in].parity * ((pi.l2 & 1) ? -1 : 1);
        if (par != irreps_out[q.i_out].parity) {
            set_error("plan: path %d violates the parity rule", p);
            return E3_ERR_BAD_PATH;
        }
        pi.in_off = in_off[q.i_in]; pi.out_off = out_off[q.i_out];
        pi.nzM = 0;
        pl.paths.push_back(pi);
        triples.push_back(pi.l1); triples.push_back(pi.l2); triples.push_back(pi.l3);
    }
    // dense CG tensors: device planner kernel (product path) or host instantiation (build check only)
    std::vector<std::vector<double>> dense;
    if (cg_on_device) {
        int rc = launch_cg_planner(triples.data(), n_paths, dense);
        if (rc != E3_OK) return rc;
    } else {
        dense.resize(n_paths);
        for (int p = 0; p < n_paths; ++p) {
            const PathInfo &pi = pl.paths[p];
            for (int a = 0; a <= 2 * pi.l1; ++a)
                for (int b = 0; b <= 2 * pi.l2; ++b)
                    for (int c = 0; c <= 2 * pi.l3; ++c) dense[p].push_back(cg_real_host(pi.l1, pi.l2, pi.l3, a, b, c));
        }
    }
    pl.nnz_total = 0;
    for (int p = 0; p < n_paths; ++p) {
        PathInfo &pi = pl.paths[p];
        int d2 = 2 * pi.l2 + 1, d3 = 2 * pi.l3 + 1;
        std::vector<char> pair((2 * pi.l1 + 1) * d3, 0);
        for (int a = 0; a <= 2 * pi.l1; ++a)
            for (int b = 0; b < d2; ++b)
                for (int c = 0; c < d3; ++c) {
                    double v = dense[p][(a * d2 + b) * d3 + c];
                    if (std::fabs(v) > 1e-12) {
                        pi.nz.push_back({ a, b, c, v });
                        pair[a * d3 + c] = 1;
                    }
                }
        for (char f : pair) pi.nzM += f;
        pl.nnz_total += (int)pi.nz.size();
    }
    return E3_OK;
}

// ---------------------------------------------------------------------------------------------
// NEXT-4 (NequIP's `64x0e + 64x0o + 32x1o + 32x1e + 32x2e + 32x2o`): per-irrep multiplicities.
// A channelwise (uvu) path keeps the multiplicity of its input irrep, so the plan falls apart into MULTIPLICITY CLASSES that
// share nothing but the edge's SH row: the composite holds one regular generated sub-plan per class, whose kernels address the
// rows of the whole plan (block offsets and row strides overridden).  Layout (the oracle's orc_tp_mul_*): a node row is the
// irrep blocks back to back, block i = (2l_i+1) x mul_i with index m*mul_i + u; a weights row is mul(p) values per path, paths
// back to back.
// ---------------------------------------------------------------------------------------------
bool plan_is_composite(const e3_irrep *irreps_in, int n_in, const e3_irrep *irreps_out, int n_out)
{
    if (!irreps_in || !irreps_out || n_in < 1 || n_out < 1) return false;
    for (int i = 0; i < n_in; ++i) if (irreps_in[i].mul != irreps_in[0].mul) return true;
    for (int i = 0; i < n_out; ++i) if (irreps_out[i].mul != irreps_in[0].mul) return true;
    return false;
}

int plan_build_composite(e3_plan &pl, const e3_irrep *irreps_in, int n_in, int sh_lmax, const e3_irrep *irreps_out, int n_out,
                         const e3_path *paths, int n_paths, e3_dtype dtype, bool cg_on_device)
{
    if (!irreps_in || !irreps_out || !paths || n_in < 1 || n_out < 1 || n_paths < 1) {
        set_error("plan: null or empty irreps / path table");
        return E3_ERR_INVALID_ARG;
    }
    if (dtype != E3_F32 && dtype != E3_BF16) { set_error("plan: unknown dtype %d", (int)dtype); return E3_ERR_INVALID_ARG; }
    if (sh_lmax < 0 || sh_lmax > kMaxL) { set_error("plan: sh_lmax %d not in 0..%d", sh_lmax, kMaxL); return E3_ERR_UNSUPPORTED; }
    pl.irreps_in.assign(irreps_in, irreps_in + n_in);
    pl.irreps_out.assign(irreps_out, irreps_out + n_out);
    pl.sh_lmax = sh_lmax;
    pl.sh_dim = (sh_lmax + 1) * (sh_lmax + 1);
    pl.dtype = dtype;
    pl.C = 0;
    std::vector<int> in_base(n_in), out_base(n_out), w_base(n_paths);
    pl.in_dim = pl.out_dim = 0;
    pl.in_size_all = pl.out_size_all = pl.w_size_all = 0;
    auto check = [&](const e3_irrep &r, const char *what, int i) {
        if (r.l < 0 || (r.parity != 1 && r.parity != -1) || r.mul < 1) { set_error("plan: bad %s irrep %d", what, i); return (int)E3_ERR_INVALID_ARG; }
        if (r.l > kMaxL) { set_error("plan: %s irrep %d has l=%d > %d", what, i, r.l, kMaxL); return (int)E3_ERR_UNSUPPORTED; }
        if (r.mul % 4 != 0) { set_error("plan: unequal multiplicities must all be multiples of 4 (%s irrep %d has %d)", what, i, r.mul); return (int)E3_ERR_UNSUPPORTED; }
        return (int)E3_OK;
    };
    for (int i = 0; i < n_in; ++i) {
        if (int rc = check(irreps_in[i], "input", i)) return rc;
        in_base[i] = pl.in_size_all;
        pl.in_size_all += (2 * irreps_in[i].l + 1) * irreps_in[i].mul;
        pl.in_dim += 2 * irreps_in[i].l + 1;
    }
    for (int i = 0; i < n_out; ++i) {
        if (int rc = check(irreps_out[i], "output", i)) return rc;
        out_base[i] = pl.out_size_all;
        pl.out_size_all += (2 * irreps_out[i].l + 1) * irreps_out[i].mul;
        pl.out_dim += 2 * irreps_out[i].l + 1;
    }
    std::vector<char> in_used(n_in, 0), out_fed(n_out, 0);
    std::vector<int> classes;                       // multiplicities in order of first use by a path
    for (int p = 0; p < n_paths; ++p) {
        const e3_path &q = paths[p];
        if (q.i_in < 0 || q.i_in >= n_in || q.i_out < 0 || q.i_out >= n_out || q.l_sh < 0 || q.l_sh > sh_lmax) {
            set_error("plan: path %d has an index out of range", p);
            return E3_ERR_BAD_PATH;
        }
        const int mul = irreps_in[q.i_in].mul;
        if (irreps_out[q.i_out].mul != mul) {
            set_error("plan: path %d joins an input irrep of multiplicity %d to an output irrep of multiplicity %d (a channelwise path keeps it)", p, mul, irreps_out[q.i_out].mul);
            return E3_ERR_BAD_PATH;
        }
        w_base[p] = pl.w_size_all;
        pl.w_size_all += mul;
        in_used[q.i_in] = 1; out_fed[q.i_out] = 1;
        if (std::find(classes.begin(), classes.end(), mul) == classes.end()) classes.push_back(mul);
    }
    pl.path_map.assign(n_paths, { 0, 0 });
    for (size_t k = 0; k < classes.size(); ++k) {
        const int mul = classes[k];
        std::vector<e3_irrep> ii, io;
        std::vector<int> gi, go;                    // sub-plan index -> index in the whole plan
        std::vector<int> li(n_in, -1), lo(n_out, -1);
        for (int i = 0; i < n_in; ++i) if (irreps_in[i].mul == mul && in_used[i]) { li[i] = (int)ii.size(); ii.push_back(irreps_in[i]); gi.push_back(i); }
        // output blocks of this multiplicity that no path feeds are still written (zeros) by this class
        for (int i = 0; i < n_out; ++i) if (irreps_out[i].mul == mul) { lo[i] = (int)io.size(); io.push_back(irreps_out[i]); go.push_back(i); out_fed[i] = 1; }
        std::vector<e3_path> pp;
        std::vector<int> gp;
        for (int p = 0; p < n_paths; ++p)
            if (irreps_in[paths[p].i_in].mul == mul) {
                pl.path_map[p] = { (int)k, (int)pp.size() };
                pp.push_back({ li[paths[p].i_in], paths[p].l_sh, lo[paths[p].i_out] });
                gp.push_back(p);
            }
        e3_plan *sp = new (std::nothrow) e3_plan();
        if (!sp) { set_error("out of host memory"); return E3_ERR_INVALID_ARG; }
        pl.subs.push_back(sp);
        int rc = plan_build_tables(*sp, ii.data(), (int)ii.size(), sh_lmax, io.data(), (int)io.size(), pp.data(), (int)pp.size(), dtype, cg_on_device);
        if (rc != E3_OK) return rc;
        sp->in_stride = pl.in_size_all; sp->out_stride = pl.out_size_all; sp->w_stride = pl.w_size_all;
        for (int g : gi) sp->in_base.push_back(in_base[g]);
        for (int g : go) sp->out_base.push_back(out_base[g]);
        for (int g : gp) sp->w_base.push_back(w_base[g]);
        pl.nnz_total += sp->nnz_total;
    }
    for (int i = 0; i < n_out; ++i)
        if (!out_fed[i]) { set_error("plan: output irrep %d is fed by no path and no multiplicity class matches it", i); return E3_ERR_UNSUPPORTED; }
    // input irreps no path reads: their rows of the per-edge grad_feats workspace are zeroed by the first class's backward
    for (int i = 0; i < n_in; ++i)
        if (!in_used[i]) pl.subs[0]->zero_in.push_back({ in_base[i], (2 * irreps_in[i].l + 1) * irreps_in[i].mul });
    // the caller's path list, for e3_plan_get_cg / counting
    pl.paths.clear();
    for (int p = 0; p < n_paths; ++p) pl.paths.push_back(pl.subs[pl.path_map[p].first]->paths[pl.path_map[p].second]);
    return E3_OK;
}

// ---------------------------------------------------------------------------------------------
// Forward roles: contiguous groups of output irreps (ordered by their first feeding path), each
// owned by one warp.  Paths that add into the same output irrep (A6) always share a role.
// ---------------------------------------------------------------------------------------------
void plan_make_roles(e3_plan &pl)
{
    const int n_out = (int)pl.irreps_out.size();
    std::vector<std::vector<int>> feeding(n_out);
    std::vector<int> first(n_out, 1 << 30);
    std::map<std::pair<int, int>, int> group_count;   // (i_in, l2) -> #paths
    for (int p = 0; p < (int)pl.paths.size(); ++p) {
        feeding[pl.paths[p].i_out].push_back(p);
        first[pl.paths[p].i_out] = std::min(first[pl.paths[p].i_out], p);
        group_count[{ pl.paths[p].i_in, pl.paths[p].l_sh }]++;
    }
    std::vector<int> order;
    for (int o = 0; o < n_out; ++o) if (!feeding[o].empty()) order.push_back(o);
    std::sort(order.begin(), order.end(), [&](int a, int b) { return first[a] < first[b]; });
    for (int o = 0; o < n_out; ++o) if (feeding[o].empty()) order.push_back(o);   // unfed blocks are still written (zeros)
    std::vector<double> cost(n_out, 0.0);
    double total_cost = 0.0;
    int total_rows = 0;
    for (int o : order) {
        for (int p : feeding[o]) {
            const PathInfo &pi = pl.paths[p];
            cost[o] += (double)pi.nz.size() + (2 * pi.l3 + 1)
                       + (double)((2 * pi.l1 + 1) * (2 * pi.l2 + 1)) / group_count[{ pi.i_in, pi.l_sh }];
        }
        total_cost += cost[o];
        total_rows += 2 * pl.irreps_out[o].l + 1;
    }
    // tuning aid: E3_TUNE="key=value,..." overrides launch-shape heuristics (never changes results).  The string is
    // tokenised on ',' and whole keys are matched (so "bwd_v2=0" does not also set "v2"); the last occurrence wins.
    const char *tune = getenv("E3_TUNE");
    std::map<std::string, int> tune_map;
    if (tune) {
        std::string t(tune);
        size_t a = 0;
        while (a <= t.size()) {
            size_t b = t.find(',', a);
            if (b == std::string::npos) b = t.size();
            std::string tok = t.substr(a, b - a);
            size_t eq = tok.find('=');
            if (eq != std::string::npos && eq > 0) tune_map[tok.substr(0, eq)] = atoi(tok.c_str() + eq + 1);
            a = b + 1;
        }
    }
    auto tune_get = [&](const char *key, int &dst) {
        auto it = tune_map.find(key);
        if (it != tune_map.end()) dst = it->second;
    };
    pl.v2 = v2_eligible(pl) ? 1 : 0;
    { int v2 = 1; tune_get("v2", v2); if (!v2) pl.v2 = 0; }
    int rows_target = 20, rows_hard = pl.v2 ? 22 : 28;
    tune_get("rows", rows_target); tune_get("rows_hard", rows_hard);
    if (rows_hard < rows_target) rows_hard = rows_target + 8;
    int n_roles = std::max(1, (total_rows + rows_target - 1) / rows_target);
    pl.roles.clear();
    Role cur; cur.rows = 0; cur.cost = 0.0;
    double cum = 0.0;
    for (size_t k = 0; k < order.size(); ++k) {
        int o = order[k];
        int r = 2 * pl.irreps_out[o].l + 1;
        bool close = !cur.out_irreps.empty() &&
                     (cur.rows + r > rows_hard ||
                      ((int)pl.roles.size() < n_roles - 1 && cum + 0.5 * cost[o] > total_cost * (pl.roles.size() + 1) / n_roles));
        if (close) { pl.roles.push_back(cur); cur = Role(); cur.rows = 0; cur.cost = 0.0; }
        cur.out_irreps.push_back(o);
        for (int p : feeding[o]) cur.paths.push_back(p);
        cur.rows += r; cur.cost += cost[o];
        cum += cost[o];
    }
    if (!cur.out_irreps.empty()) pl.roles.push_back(cur);
    for (Role &ro : pl.roles) std::sort(ro.paths.begin(), ro.paths.end());
    // channels per lane / channel blocks
    pl.K = (pl.C % 64 == 0) ? 2 : 1;
    pl.nchb = (pl.C + 32 * pl.K - 1) / (32 * pl.K);
    const int slot_bytes = pl.K * (pl.dtype == E3_BF16 ? 2 : 4);
    // rings need 4/8-byte lane slots and 4-byte granular SH rows (bf16 with an odd sh_dim falls back to plain loads)
    pl.ring = (pl.C % (32 * pl.K) == 0) && (slot_bytes == 4 || slot_bytes == 8) &&
              ((pl.sh_dim * (pl.dtype == E3_BF16 ? 2 : 4)) % 4 == 0);
    // forward ring depth: roles with long per-edge bodies hide the load latency with fewer stages in
    // flight (and a shallower ring leaves room for more resident CTAs)
    pl.fwd_depth = (total_cost / std::max<size_t>(1, pl.roles.size()) >= 100.0) ? 2 : 4;
    pl.fwd_minb = 4;
    pl.bwd_minb = 3;           // gen_backward_source lowers it when the shared-memory footprint allows fewer CTAs
    if (pl.v2) {               // second-generation kernels: 4 channels per lane, EPS edges per warp step
        pl.lpe = pl.C >= 128 ? 32 : pl.C / 4;
        pl.eps = 32 / pl.lpe;
        pl.nchb2 = pl.C >= 128 ? pl.C / 128 : 1;
        pl.fwd_depth = pl.eps >= 2 ? 2 : 3;
        pl.fwd_minb = 3;
        pl.bwd_v2 = 1;
        pl.bwd_minb = 2;
    }
    tune_get("bwd_v2", pl.bwd_v2); tune_get("fwd_depth_max", pl.fwd_depth_max); tune_get("bwd_depth", pl.bwd_depth); tune_get("bwd_role_cost", pl.bwd_role_cost); tune_get("bwd_chunk", pl.bwd_chunk); tune_get("bwd_r", pl.bwd_r); tune_get("bwd_split", pl.bwd_split); tune_get("fwd_split", pl.fwd_split);
    if (!pl.v2) pl.bwd_v2 = 0;
    tune_get("fwd_minb", pl.fwd_minb); tune_get("bwd_minb", pl.bwd_minb);
    tune_get("fwd_warps", pl.fwd_warps); tune_get("bwd_warps", pl.bwd_warps);
    tune_get("fwd_depth", pl.fwd_depth); tune_get("chunk", pl.fwd_chunk); tune_get("wait_all", pl.wait_all);
    tune_get("bwd_overlap", pl.bwd_overlap);
    // third-generation forward: roles aligned with the input irreps, grouped into teams that share one CTA and one copy of
    // the sender rows per edge
    tune_get("fwd_v3_bulk", pl.fwd_v3_bulk);
    pl.fwd_v3 = 0;             // opt-in (E3_TUNE fwd_v3=1): measured no faster than the second generation (experiment viii)
    tune_get("fwd_v3", pl.fwd_v3);
    if (!pl.v2 || !v3_eligible(pl) || !pl.in_base.empty()) pl.fwd_v3 = 0;      // the v3 generator knows the regular layout only (not the sub-plans of a composite)
    tune_get("team", pl.fwd_tw); tune_get("fwd_v3_depth", pl.fwd_v3_depth); tune_get("fwd_v3_lag", pl.fwd_v3_lag); tune_get("fwd_v3_chunk", pl.fwd_v3_chunk); tune_get("fwd_v3_bulk", pl.fwd_v3_bulk);
    pl.fwd_tw = std::max(1, std::min(4, pl.fwd_tw));
    pl.fwd_v3_lag = std::max(1, std::min(2, pl.fwd_v3_lag));
    if (pl.fwd_v3) {
        pl.roles.clear();
        pl.teams.clear();
        std::vector<std::vector<int>> groups;        // runs of output irreps fed by the same input irrep
        int last_dom = -2;
        for (int o : order) {
            const int dom = feeding[o].empty() ? -1 : pl.paths[first[o]].i_in;
            if (groups.empty() || dom != last_dom) groups.push_back({});
            groups.back().push_back(o);
            last_dom = dom;
        }
        // cost of an output irrep in packed 4-channel operations of the factored form (nzM FMAs + the weight multiply) plus its
        // scalar A entries (one FMUL / FFMA per non-zero, a quarter of a packed operation's pipe time)
        for (int o : order) {
            cost[o] = 0.0;
            for (int p : feeding[o]) {
                const PathInfo &pi = pl.paths[p];
                cost[o] += pi.nzM + std::min(2 * pi.l1 + 1, 2 * pi.l3 + 1) + 0.25 * (double)pi.nz.size();
            }
        }
        std::vector<std::vector<int>> group_roles;
        for (auto &grp : groups) {
            int rows_g = 0;
            double cost_g = 0;
            for (int o : grp) { rows_g += 2 * pl.irreps_out[o].l + 1; cost_g += cost[o]; }
            const int n_r = std::max(1, (rows_g + rows_hard - 1) / rows_hard);
            group_roles.push_back({});
            // contiguous split of the group's output irreps into n_r roles minimising the largest role cost, rows <= rows_hard
            // per role (more roles if that is infeasible): exact search, the groups are tiny
            const int n = (int)grp.size();
            std::vector<int> best_cut;
            for (int k = n_r; k <= n && best_cut.empty(); ++k) {
                double best = 1e300;
                std::vector<int> cut(k + 1, 0);
                std::function<void(int, int, double)> rec = [&](int part, int start, double worst) {
                    if (part == k - 1) {
                        int rows = 0; double c = 0;
                        for (int i = start; i < n; ++i) { rows += 2 * pl.irreps_out[grp[i]].l + 1; c += cost[grp[i]]; }
                        if (start >= n || (rows > rows_hard && n - start > 1)) return;
                        const double wv = std::max(worst, c);
                        if (wv < best) { best = wv; cut[k] = n; best_cut = cut; }
                        return;
                    }
                    int rows = 0; double c = 0;
                    for (int end = start + 1; end <= n - (k - 1 - part); ++end) {
                        rows += 2 * pl.irreps_out[grp[end - 1]].l + 1; c += cost[grp[end - 1]];
                        if (rows > rows_hard && end - start > 1) break;
                        cut[part + 1] = end;
                        rec(part + 1, end, std::max(worst, c));
                    }
                };
                rec(0, 0, 0.0);
            }
            if (best_cut.empty()) { best_cut.clear(); for (int i = 0; i <= n; ++i) best_cut.push_back(i); }
            for (size_t q = 0; q + 1 < best_cut.size(); ++q) {
                Role cur2; cur2.rows = 0; cur2.cost = 0.0;
                for (int i = best_cut[q]; i < best_cut[q + 1]; ++i) {
                    const int o2 = grp[i];
                    cur2.out_irreps.push_back(o2);
                    for (int p : feeding[o2]) cur2.paths.push_back(p);
                    cur2.rows += 2 * pl.irreps_out[o2].l + 1; cur2.cost += cost[o2];
                }
                group_roles.back().push_back((int)pl.roles.size());
                pl.roles.push_back(cur2);
            }
        }
        for (Role &ro : pl.roles) std::sort(ro.paths.begin(), ro.paths.end());
        std::vector<int> team;
        for (auto &gr : group_roles) {
            if (!team.empty() && (int)(team.size() + gr.size()) > pl.fwd_tw) { pl.teams.push_back(team); team.clear(); }
            for (int ri : gr) {
                if ((int)team.size() == pl.fwd_tw) { pl.teams.push_back(team); team.clear(); }
                team.push_back(ri);
            }
        }
        if (!team.empty()) pl.teams.push_back(team);
    }
}

}  // namespace e3

// ---------------------------------------------------------------------------------------------
// C ABI: path enumeration helper (host only)
// ---------------------------------------------------------------------------------------------
extern "C" int e3_all_paths(const e3_irrep *irreps_in, int n_in, int sh_lmax, int out_lmax, int natural_parity_only,
                            e3_irrep *irreps_out, int *n_out, e3_path *paths, int *n_paths)
{
    if (!irreps_in || n_in < 1 || !n_out || !n_paths || sh_lmax < 0 || out_lmax < 0) {
        e3::set_error("e3_all_paths: bad arguments");
        return E3_ERR_INVALID_ARG;
    }
    int cap_out = *n_out, cap_paths = *n_paths, n = 0;
    for (int i = 0; i < n_in; ++i) {
        int l1 = irreps_in[i].l, p1 = irreps_in[i].parity;
        for (int l2 = 0; l2 <= sh_lmax; ++l2) {
            int lo = l1 > l2 ? l1 - l2 : l2 - l1;
            int hi = l1 + l2 < out_lmax ? l1 + l2 : out_lmax;
            for (int l3 = lo; l3 <= hi; ++l3) {
                int p3 = p1 * ((l2 & 1) ? -1 : 1);
                if (natural_parity_only && p3 != ((l3 & 1) ? -1 : 1)) continue;
                if (irreps_out && paths) {
                    if (n >= cap_out || n >= cap_paths) { e3::set_error("e3_all_paths: output arrays too small"); return E3_ERR_INVALID_ARG; }
                    irreps_out[n] = { l3, p3, irreps_in[i].mul };
                    paths[n] = { i, l2, n };
                }
                ++n;
            }
        }
    }
    *n_out = n;
    *n_paths = n;
    return E3_OK;
}
