// NEXT-3: MACE's symmetric contraction at correlation order 2 on node features, the other operation the paper routes
// to e3j (PAPER.md L535 `node_symmetry 2`, L536 `correlation 2`, L545 `symmetric_contraction_backend e3j`).  The paper prints no
// formula; reading S1: every path has one weight per species and channel, W[z, path, u], and is either
//   linear     (i_in1, -1,    i_out):  B[n, i_out, M, u] += W * A[n, i_in1, M, u]
//   quadratic  (i_in1, i_in2, i_out):  B[n, i_out, M, u] += W * sum_{m1,m2} C^{l1 l2 L}[m1,m2,M] A[n,i_in1,m1,u] A[n,i_in2,m2,u]
// with the real Clebsch-Gordan tensors of reading A4 (computed by the device planner kernel of plan.cu).
//
// This is a per-node operation (N x C independent columns, no gather, no scatter): the kernels are table-driven.  The sparse CG
// terms are flattened on the host into three CSR lists -- by OUTPUT row (forward), by INPUT row (grad_feats; a quadratic term
// appears once for each of its two factors) and by PATH (grad_weights) -- so that every result element is accumulated in a
// register by one thread in a fixed order (deterministic, no atomics).  A block owns one node and up to 128 channels; the node's
// feature row (and cotangent row) is staged in shared memory.  grad_weights is a sum over the nodes of a species: per-chunk
// partial sums (about 32 nodes per chunk) written by one thread per (path, channel), added in chunk order by a second kernel.
// These table-driven kernels are the FALLBACK: by default e3_symcon_create generates the three kernels for the path table at run
// time (gen_symcon_source below: rows in registers, CG coefficients as immediates, shared products), 8x / 6x faster on a
// 100 000-node, 64-channel, l <= 3 case (forward 2.95 -> 0.36 ms = 0.99 of the HBM roofline; VJP 8.1 -> 1.36 ms).
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <map>
#include <new>
#include <string>
#include <vector>

#include "e3_internal.h"

using namespace e3;

struct e3_symcon {
    int n_in = 0, n_out = 0, n_paths = 0, n_species = 0, C = 0, in_dim = 0, out_dim = 0, nnz = 0;
    // device tables
    int *f_ptr = nullptr, *f_a1 = nullptr, *f_a2 = nullptr, *f_p = nullptr; float *f_c = nullptr;          // by output row
    int *b_ptr = nullptr, *b_other = nullptr, *b_g = nullptr, *b_p = nullptr; float *b_c = nullptr;       // by input row
    int *w_ptr = nullptr, *w_a1 = nullptr, *w_a2 = nullptr, *w_g = nullptr; float *w_c = nullptr;         // by path
    // run-time specialised kernels (the CG terms as straight-line code with immediate coefficients, rows in registers); the table-driven
    // kernels above stay as the fallback for very long term lists and for E3_SYMCON_JIT=0
    bool jit = false;
    e3::JitKernel jfwd, jbf, jbw, jbb;
    int acc_smem = 0;      // bytes of the node-chunk kernels' shared accumulators (n_species * n_paths * 128 floats); 0 = too large, table-driven grad_weights
    int slots = 0;         // CTAs of e3_sc_bwd_both resident on the device at once (the chunk count is rounded to whole waves of them)
};

namespace {

// node chunks of the grad_weights partial sums: a thread (chunk, channel) walks its chunk's nodes serially.  At most 128 nodes per chunk;
// the number of 128-thread CTAs is rounded up to whole waves of `slots` resident CTAs (equal-length CTAs: a partial last wave costs a
// whole one; measured on 100 000 nodes x 64 channels: one wave of 85-node chunks 0.50 ms, three waves of 29-node chunks 0.52, five of 15
// 0.54); small problems get shorter chunks (down to 4 nodes) so that the launch still covers the machine; at most 256 MB of partial
// sums.  A function of (N, C, table sizes, device) only: the summation order is fixed for a given problem on a given device type.
static int symcon_chunks(long long N, long long C, long long per_chunk_floats, long long slots)
{
    if (N <= 0) return 1;
    if (C < 1) C = 1;
    if (slots < 1) slots = 592;
    long long c = (N + 127) / 128;
    long long ctas = (c * C + 127) / 128;
    if (ctas < slots) {                                   // small problem: shorter chunks, one wave at most
        const long long c4 = (N + 3) / 4, ctas4 = (c4 * C + 127) / 128;
        ctas = ctas4 < slots ? ctas4 : slots;
    } else {
        ctas = ((ctas + slots - 1) / slots) * slots;
    }
    c = (ctas * 128) / C;
    if (c < 1) c = 1;
    if (c > N) c = N;
    const long long cap = (256LL << 20) / 4 / (per_chunk_floats > 0 ? per_chunk_floats : 1);
    if (c > cap) c = cap < 1 ? 1 : cap;
    return (int)c;
}

__global__ void symcon_fwd_kernel(const float *__restrict__ A, const int32_t *__restrict__ species, const float *__restrict__ W, int C, int in_dim,
                                  int out_dim, int n_paths, int n_species, const int *__restrict__ ptr, const int *__restrict__ a1, const int *__restrict__ a2,
                                  const int *__restrict__ tp, const float *__restrict__ tc, float *__restrict__ B)
{
    extern __shared__ float As[];                      // [in_dim][CB]
    const int n = blockIdx.x, CB = blockDim.x, u = blockIdx.y * CB + threadIdx.x;
    const bool act = u < C;
    for (int r = 0; r < in_dim; ++r) As[r * CB + threadIdx.x] = act ? A[((size_t)n * in_dim + r) * C + u] : 0.0f;
    int z = species[n];
    z = z < 0 ? 0 : (z >= n_species ? n_species - 1 : z);      // range is checked by the entry point's caller contract; clamp, never read out of bounds
    if (!act) return;
    const float *Wz = W + (size_t)z * n_paths * C + u;
    for (int R = 0; R < out_dim; ++R) {
        float acc = 0.0f;
        for (int t = ptr[R]; t < ptr[R + 1]; ++t) {
            const float w = __ldg(Wz + (size_t)tp[t] * C);
            const float x1 = As[a1[t] * CB + threadIdx.x];
            const int j = a2[t];
            acc = fmaf(w * tc[t], j >= 0 ? x1 * As[j * CB + threadIdx.x] : x1, acc);
        }
        B[((size_t)n * out_dim + R) * C + u] = acc;
    }
}

__global__ void symcon_bwd_feats_kernel(const float *__restrict__ A, const int32_t *__restrict__ species, const float *__restrict__ W, const float *__restrict__ G,
                                        int C, int in_dim, int out_dim, int n_paths, int n_species, const int *__restrict__ ptr, const int *__restrict__ other,
                                        const int *__restrict__ grow, const int *__restrict__ tp, const float *__restrict__ tc, float *__restrict__ dA)
{
    extern __shared__ float sm[];                      // A [in_dim][CB] then G [out_dim][CB]
    const int n = blockIdx.x, CB = blockDim.x, u = blockIdx.y * CB + threadIdx.x;
    float *As = sm, *Gs = sm + in_dim * CB;
    const bool act = u < C;
    for (int r = 0; r < in_dim; ++r) As[r * CB + threadIdx.x] = act ? A[((size_t)n * in_dim + r) * C + u] : 0.0f;
    for (int r = 0; r < out_dim; ++r) Gs[r * CB + threadIdx.x] = act ? G[((size_t)n * out_dim + r) * C + u] : 0.0f;
    int z = species[n];
    z = z < 0 ? 0 : (z >= n_species ? n_species - 1 : z);
    if (!act) return;
    const float *Wz = W + (size_t)z * n_paths * C + u;
    for (int R = 0; R < in_dim; ++R) {
        float acc = 0.0f;
        for (int t = ptr[R]; t < ptr[R + 1]; ++t) {
            const float w = __ldg(Wz + (size_t)tp[t] * C);
            const float g = Gs[grow[t] * CB + threadIdx.x];
            const int j = other[t];
            acc = fmaf(w * tc[t], j >= 0 ? g * As[j * CB + threadIdx.x] : g, acc);
        }
        dA[((size_t)n * in_dim + R) * C + u] = acc;
    }
}

// grid (chunks, ceil(n_paths * C / 128)): thread = (path, channel); partial[chunk][species][path][channel] over the chunk's nodes in ascending order
__global__ void symcon_bwd_w_partial_kernel(const float *__restrict__ A, const int32_t *__restrict__ species, const float *__restrict__ G, int C, int in_dim,
                                            int out_dim, int n_paths, int n_species, int N, int n_chunks, const int *__restrict__ ptr, const int *__restrict__ a1,
                                            const int *__restrict__ a2, const int *__restrict__ grow, const float *__restrict__ tc, float *__restrict__ partial)
{
    const int idx = blockIdx.y * blockDim.x + threadIdx.x;
    if (idx >= n_paths * C) return;
    const int p = idx / C, u = idx % C;
    const int per = (N + n_chunks - 1) / n_chunks, n0 = min(N, (int)blockIdx.x * per), n1 = min(N, n0 + per);
    float *dst = partial + (size_t)blockIdx.x * n_species * n_paths * C + idx;
    for (int s = 0; s < n_species; ++s) dst[(size_t)s * n_paths * C] = 0.0f;
    const int t0 = ptr[p], t1 = ptr[p + 1];
    for (int n = n0; n < n1; ++n) {
        const float *a = A + (size_t)n * in_dim * C + u, *g = G + (size_t)n * out_dim * C + u;
        float acc = 0.0f;
        for (int t = t0; t < t1; ++t) {
            const float x1 = a[(size_t)a1[t] * C];
            const int j = a2[t];
            acc = fmaf(tc[t] * g[(size_t)grow[t] * C], j >= 0 ? x1 * a[(size_t)j * C] : x1, acc);
        }
        int z = species[n];
        z = z < 0 ? 0 : (z >= n_species ? n_species - 1 : z);
        dst[(size_t)z * n_paths * C] += acc;
    }
}

// dW[i] = sum over the chunks of partial[chunk][i]: block = 32 outputs x 32 chunk lanes; lane y adds chunks y, y+32, ... in ascending
// order, the 32 lane sums are added in lane order (fixed order: deterministic)
__global__ void __launch_bounds__(1024) symcon_bwd_w_reduce_kernel(const float *__restrict__ partial, int total, int n_chunks, float *__restrict__ dW)
{
    __shared__ float part[32][33];
    const int i = blockIdx.x * 32 + threadIdx.x;
    float acc = 0.0f;
    if (i < total)
        for (int c = threadIdx.y; c < n_chunks; c += 32) acc += partial[(size_t)c * total + i];
    part[threadIdx.y][threadIdx.x] = acc;
    __syncthreads();
    if (threadIdx.y == 0 && i < total) {
        float t = 0.0f;
#pragma unroll
        for (int y = 0; y < 32; ++y) t += part[y][threadIdx.x];
        dW[i] = t;
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// Run-time specialisation (same idea as the tensor-product kernels): one thread = one (node, channel); the node's input rows
// (and, for grad_feats, its cotangent rows) live in registers, every CG term is an FMUL / FFMA with an immediate coefficient,
// products x[a1] * x[a2] are shared between the terms that use them.  grad_weights: one thread = one (node chunk, channel),
// per path s_p = sum_R g[R] * (sum of the row's terms), added to the chunk's partial sums.
// ---------------------------------------------------------------------------------------------------------------------
struct ScTerm { int a1, a2, grow, p; float c; };

struct Gen {
    std::string s;
    void f(const char *fmt, ...)
    {
        char buf[1024];
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(buf, sizeof(buf), fmt, ap);
        va_end(ap);
        s += buf;
    }
};

std::string fimm(float c)
{
    char b[64];
    snprintf(b, sizeof(b), "%.9g", (double)c);
    std::string t(b);
    if (t.find('.') == std::string::npos && t.find('e') == std::string::npos && t.find("inf") == std::string::npos) t += ".0";
    return t + "f";
}

// emits (once) and names the product of a term's input rows
std::string sc_prod(Gen &o, std::map<std::pair<int, int>, int> &seen, const ScTerm &t, const char *ind)
{
    if (t.a2 < 0) return "x" + std::to_string(t.a1);
    const int a = std::min(t.a1, t.a2), b = std::max(t.a1, t.a2);
    if (!seen.count({ a, b })) {
        seen[{ a, b }] = 1;
        o.f("%sconst float q%d_%d = x%d * x%d;\n", ind, a, b, a, b);
    }
    return "q" + std::to_string(a) + "_" + std::to_string(b);
}

// sum of a row's terms of one path as an expression tree of fmaf's; returns the name of the temporary holding it
std::string sc_row_sum(Gen &o, std::map<std::pair<int, int>, int> &seen, const std::vector<ScTerm> &ts, int R, int p, const char *ind, int &tmp)
{
    std::string acc;
    for (const ScTerm &t : ts) {
        if (t.grow != R || t.p != p) continue;
        const std::string pr = sc_prod(o, seen, t, ind);
        const std::string nm = "r" + std::to_string(tmp++);
        if (acc.empty()) o.f("%sconst float %s = %s * %s;\n", ind, nm.c_str(), fimm(t.c).c_str(), pr.c_str());
        else o.f("%sconst float %s = fmaf(%s, %s, %s);\n", ind, nm.c_str(), fimm(t.c).c_str(), pr.c_str(), acc.c_str());
        acc = nm;
    }
    return acc;
}

std::string gen_symcon_source(const std::vector<ScTerm> &ts, int in_dim, int out_dim, int n_paths)
{
    Gen o;
    o.f("// generated by libe3b200: symmetric contraction, %d CG terms, %d input rows, %d output rows, %d paths\n", (int)ts.size(), in_dim, out_dim, n_paths);
    o.f("#define IN %d\n#define OUT %d\n#define NP %d\n", in_dim, out_dim, n_paths);
    // (row, path) pairs that carry terms, in row order
    std::vector<std::pair<int, int>> rp;
    for (int R = 0; R < out_dim; ++R)
        for (int p = 0; p < n_paths; ++p) {
            bool any = false;
            for (const ScTerm &t : ts) any = any || (t.grow == R && t.p == p);
            if (any) rp.push_back({ R, p });
        }
    const char *head = "  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;\n  if (idx >= NC) return;\n"
                       "  const long long n = idx / C;\n  const int u = (int)(idx - n * C);\n"
                       "  const float *a = A + (size_t)n * IN * C + u;\n";
    // ---- forward
    o.f("extern \"C\" __global__ void __launch_bounds__(128) e3_sc_fwd(const float *__restrict__ A, const int *__restrict__ species, const float *__restrict__ W,\n"
        "    long long NC, int C, int n_species, float *__restrict__ B)\n{\n%s", head);
    for (int r = 0; r < in_dim; ++r) o.f("  const float x%d = a[(size_t)%d * C];\n", r, r);
    o.f("  int z = species[n]; z = z < 0 ? 0 : (z >= n_species ? n_species - 1 : z);\n"
        "  const float *w = W + (size_t)z * NP * C + u;\n  float *b = B + (size_t)n * OUT * C + u;\n");
    for (int p = 0; p < n_paths; ++p) o.f("  const float w%d = w[(size_t)%d * C];\n", p, p);
    {
        std::map<std::pair<int, int>, int> seen;
        int tmp = 0;
        for (int R = 0; R < out_dim; ++R) {
            std::string total;
            for (auto &q : rp) {
                if (q.first != R) continue;
                const std::string sum = sc_row_sum(o, seen, ts, R, q.second, "  ", tmp);
                const std::string nm = "o" + std::to_string(tmp++);
                if (total.empty()) o.f("  const float %s = w%d * %s;\n", nm.c_str(), q.second, sum.c_str());
                else o.f("  const float %s = fmaf(w%d, %s, %s);\n", nm.c_str(), q.second, sum.c_str(), total.c_str());
                total = nm;
            }
            o.f("  b[(size_t)%d * C] = %s;\n", R, total.empty() ? "0.0f" : total.c_str());
        }
    }
    o.f("}\n\n");
    // ---- grad_feats
    o.f("extern \"C\" __global__ void __launch_bounds__(128) e3_sc_bwd_feats(const float *__restrict__ A, const int *__restrict__ species, const float *__restrict__ W,\n"
        "    const float *__restrict__ G, long long NC, int C, int n_species, float *__restrict__ dA)\n{\n%s", head);
    for (int r = 0; r < in_dim; ++r) o.f("  const float x%d = a[(size_t)%d * C]; float d%d = 0.0f;\n", r, r, r);
    o.f("  int z = species[n]; z = z < 0 ? 0 : (z >= n_species ? n_species - 1 : z);\n"
        "  const float *w = W + (size_t)z * NP * C + u;\n  const float *g = G + (size_t)n * OUT * C + u;\n");
    for (int p = 0; p < n_paths; ++p) o.f("  const float w%d = w[(size_t)%d * C];\n", p, p);
    for (auto &q : rp) {
        o.f("  { const float gw = w%d * g[(size_t)%d * C];\n", q.second, q.first);
        for (const ScTerm &t : ts) {
            if (t.grow != q.first || t.p != q.second) continue;
            if (t.a2 < 0) { o.f("    d%d = fmaf(%s, gw, d%d);\n", t.a1, fimm(t.c).c_str(), t.a1); continue; }
            o.f("    { const float cg = %s * gw; d%d = fmaf(cg, x%d, d%d); d%d = fmaf(cg, x%d, d%d); }\n", fimm(t.c).c_str(), t.a1, t.a2, t.a1, t.a2, t.a1, t.a2);
        }
        o.f("  }\n");
    }
    o.f("  float *da = dA + (size_t)n * IN * C + u;\n");
    for (int r = 0; r < in_dim; ++r) o.f("  da[(size_t)%d * C] = d%d;\n", r, r);
    o.f("}\n\n");
    // ---- node-chunk kernels: thread = (chunk, channel) walks the chunk's nodes in ascending order; the grad_weights contributions
    // s_p = sum_R g[R] * (row sum) are added to per-thread accumulators [species][path] in shared memory (column threadIdx.x of a
    // [n_species * NP][128] array: no bank conflicts, no sharing between threads) and written out once per chunk.  e3_sc_bwd_w does only
    // that; e3_sc_bwd_both also forms the node's grad_feats rows (same statements, same order as e3_sc_bwd_feats), so that a VJP call
    // that wants both gradients reads feats and grad_out once.
    for (int both = 0; both < 2; ++both) {
        o.f("extern \"C\" __global__ void __launch_bounds__(128, 4) %s(const float *__restrict__ A, const int *__restrict__ species, const float *__restrict__ W,\n"
            "    const float *__restrict__ G, int N, int C, int n_species, int n_chunks, float *__restrict__ dA, float *__restrict__ partial)\n{\n",
            both ? "e3_sc_bwd_both" : "e3_sc_bwd_w");
        o.s += "  extern __shared__ float acc[];\n"
               "  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;\n  if (idx >= (long long)n_chunks * C) return;\n"
               "  const int chunk = (int)(idx / C), u = (int)(idx - (long long)chunk * C);\n"
               "  const int per = (N + n_chunks - 1) / n_chunks;\n  const int n0 = min(N, chunk * per), n1 = min(N, n0 + per);\n"
               "  float *my = acc + threadIdx.x;\n  const int nacc = n_species * NP;\n"
               "  for (int i = 0; i < nacc; ++i) my[i * 128] = 0.0f;\n"
               "#pragma unroll 1\n  for (int n = n0; n < n1; ++n) {\n"
               "    const float *a = A + (size_t)n * IN * C + u, *g = G + (size_t)n * OUT * C + u;\n";
        for (int r = 0; r < in_dim; ++r) o.f(both ? "    const float x%d = a[(size_t)%d * C]; float d%d = 0.0f;\n" : "    const float x%d = a[(size_t)%d * C];\n", r, r, r);
        o.f("    int z = species[n]; z = z < 0 ? 0 : (z >= n_species ? n_species - 1 : z);\n    float *mz = my + z * NP * 128;\n");
        if (both) {
            o.f("    const float *w = W + (size_t)z * NP * C + u;\n");
            for (int p = 0; p < n_paths; ++p) o.f("    const float w%d = w[(size_t)%d * C];\n", p, p);
        }
        std::map<std::pair<int, int>, int> seen;
        std::vector<std::string> cur(n_paths);
        int tmp = 0, k = 0;
        for (auto &q : rp) {                                           // row-major, as in e3_sc_bwd_feats; per path the rows ascend
            o.f("    const float g%d = g[(size_t)%d * C];\n", k, q.first);
            const std::string sum = sc_row_sum(o, seen, ts, q.first, q.second, "    ", tmp);
            const std::string nm = "s" + std::to_string(tmp++);
            if (cur[q.second].empty()) o.f("    const float %s = g%d * %s;\n", nm.c_str(), k, sum.c_str());
            else o.f("    const float %s = fmaf(g%d, %s, %s);\n", nm.c_str(), k, sum.c_str(), cur[q.second].c_str());
            cur[q.second] = nm;
            if (both) {
                o.f("    { const float gw = w%d * g%d;\n", q.second, k);
                for (const ScTerm &t : ts) {
                    if (t.grow != q.first || t.p != q.second) continue;
                    if (t.a2 < 0) { o.f("      d%d = fmaf(%s, gw, d%d);\n", t.a1, fimm(t.c).c_str(), t.a1); continue; }
                    o.f("      { const float cg = %s * gw; d%d = fmaf(cg, x%d, d%d); d%d = fmaf(cg, x%d, d%d); }\n", fimm(t.c).c_str(), t.a1, t.a2, t.a1, t.a2, t.a1, t.a2);
                }
                o.f("    }\n");
            }
            ++k;
        }
        for (int p = 0; p < n_paths; ++p)
            if (!cur[p].empty()) o.f("    mz[%d * 128] += %s;\n", p, cur[p].c_str());
        if (both) {
            o.f("    float *da = dA + (size_t)n * IN * C + u;\n");
            for (int r = 0; r < in_dim; ++r) o.f("    da[(size_t)%d * C] = d%d;\n", r, r);
        }
        o.s += "  }\n  float *dst = partial + (size_t)chunk * nacc * C + u;\n"
               "  for (int i = 0; i < nacc; ++i) dst[(size_t)i * C] = my[i * 128];\n}\n\n";
    }
    return o.s;
}

template <typename T>
int upload(T **dst, const std::vector<T> &v)
{
    const size_t b = std::max<size_t>(v.size(), 1) * sizeof(T);
    E3_CUDA_TRY(cudaMalloc((void **)dst, b));
    if (!v.empty()) E3_CUDA_TRY(cudaMemcpy(*dst, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice));
    return E3_OK;
}

}  // namespace

extern "C" int e3_symcon_destroy(e3_symcon *sc)
{
    if (!sc) return E3_OK;
    void *ptrs[] = { sc->f_ptr, sc->f_a1, sc->f_a2, sc->f_p, sc->f_c, sc->b_ptr, sc->b_other, sc->b_g, sc->b_p, sc->b_c, sc->w_ptr, sc->w_a1, sc->w_a2, sc->w_g, sc->w_c };
    for (void *p : ptrs) if (p) cudaFree(p);
    jit_unload(sc->jfwd); jit_unload(sc->jbf); jit_unload(sc->jbw); jit_unload(sc->jbb);
    delete sc;
    return E3_OK;
}

// device = false: build-time check only (host CG instantiation, generation + NVRTC compilation, nothing uploaded or loaded)
static int symcon_create_impl(e3_symcon **out, const e3_irrep *irreps_in, int n_in, const e3_irrep *irreps_out, int n_out, const e3_pair_path *paths,
                              int n_paths, int n_species, bool device, int *regs, int *spill)
{
    if (!out || !irreps_in || !irreps_out || !paths || n_in < 1 || n_out < 1 || n_paths < 1 || n_species < 1) { set_error("e3_symcon_create: bad arguments"); return E3_ERR_INVALID_ARG; }
    *out = nullptr;
    int ndev = 0;
    if (device && (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1)) { cudaGetLastError(); set_error("e3_symcon_create: no CUDA device (no CPU fallback)"); return E3_ERR_CUDA; }
    const int C = irreps_in[0].mul;
    std::vector<int> in_off(n_in), out_off(n_out);
    int in_dim = 0, out_dim = 0;
    for (int i = 0; i < n_in; ++i) {
        if (irreps_in[i].mul != C || C < 1) { set_error("symmetric contraction: all multiplicities must be equal"); return E3_ERR_UNSUPPORTED; }
        if (irreps_in[i].l < 0 || irreps_in[i].l > kMaxL || (irreps_in[i].parity != 1 && irreps_in[i].parity != -1)) { set_error("symmetric contraction: bad input irrep %d", i); return E3_ERR_UNSUPPORTED; }
        in_off[i] = in_dim; in_dim += 2 * irreps_in[i].l + 1;
    }
    for (int i = 0; i < n_out; ++i) {
        if (irreps_out[i].mul != C) { set_error("symmetric contraction: all multiplicities must be equal"); return E3_ERR_UNSUPPORTED; }
        if (irreps_out[i].l < 0 || irreps_out[i].l > kMaxL || (irreps_out[i].parity != 1 && irreps_out[i].parity != -1)) { set_error("symmetric contraction: bad output irrep %d", i); return E3_ERR_UNSUPPORTED; }
        out_off[i] = out_dim; out_dim += 2 * irreps_out[i].l + 1;
    }
    std::vector<int> triples;
    std::vector<int> quad_of(n_paths, -1);
    for (int p = 0; p < n_paths; ++p) {
        const e3_pair_path q = paths[p];
        if (q.i_in1 < 0 || q.i_in1 >= n_in || q.i_in2 >= n_in || q.i_out < 0 || q.i_out >= n_out) { set_error("symmetric contraction: path %d has an index out of range", p); return E3_ERR_BAD_PATH; }
        const int L = irreps_out[q.i_out].l;
        if (q.i_in2 < 0) {
            if (irreps_in[q.i_in1].l != L || irreps_in[q.i_in1].parity != irreps_out[q.i_out].parity) { set_error("symmetric contraction: linear path %d changes the irrep", p); return E3_ERR_BAD_PATH; }
        } else {
            const int l1 = irreps_in[q.i_in1].l, l2 = irreps_in[q.i_in2].l;
            if (L < std::abs(l1 - l2) || L > l1 + l2) { set_error("symmetric contraction: path %d violates the triangle rule", p); return E3_ERR_BAD_PATH; }
            if (irreps_in[q.i_in1].parity * irreps_in[q.i_in2].parity != irreps_out[q.i_out].parity) { set_error("symmetric contraction: path %d violates the parity rule", p); return E3_ERR_BAD_PATH; }
            quad_of[p] = (int)triples.size() / 3;
            triples.push_back(l1); triples.push_back(l2); triples.push_back(L);
        }
    }
    std::vector<std::vector<double>> dense;
    if (!triples.empty() && device) {
        int rc = launch_cg_planner(triples.data(), (int)triples.size() / 3, dense);
        if (rc != E3_OK) return rc;
    } else {
        for (size_t q = 0; q + 2 < triples.size(); q += 3) {
            const int l1 = triples[q], l2 = triples[q + 1], L = triples[q + 2];
            std::vector<double> d;
            for (int a = 0; a <= 2 * l1; ++a)
                for (int b = 0; b <= 2 * l2; ++b)
                    for (int c = 0; c <= 2 * L; ++c) d.push_back(cg_real_host(l1, l2, L, a, b, c));
            dense.push_back(d);
        }
    }
    struct Term { int a1, a2, grow, p; float c; };
    std::vector<Term> terms;
    for (int p = 0; p < n_paths; ++p) {
        const e3_pair_path q = paths[p];
        const int L = irreps_out[q.i_out].l;
        if (q.i_in2 < 0) {
            for (int M = 0; M <= 2 * L; ++M) terms.push_back({ in_off[q.i_in1] + M, -1, out_off[q.i_out] + M, p, 1.0f });
        } else {
            const int l1 = irreps_in[q.i_in1].l, l2 = irreps_in[q.i_in2].l;
            const std::vector<double> &cg = dense[quad_of[p]];
            for (int m1 = 0; m1 <= 2 * l1; ++m1)
                for (int m2 = 0; m2 <= 2 * l2; ++m2)
                    for (int M = 0; M <= 2 * L; ++M) {
                        const double c = cg[(m1 * (2 * l2 + 1) + m2) * (2 * L + 1) + M];
                        if (std::fabs(c) > 1e-12) terms.push_back({ in_off[q.i_in1] + m1, in_off[q.i_in2] + m2, out_off[q.i_out] + M, p, (float)c });
                    }
        }
    }
    e3_symcon *sc = new (std::nothrow) e3_symcon();
    if (!sc) { set_error("out of host memory"); return E3_ERR_INVALID_ARG; }
    sc->n_in = n_in; sc->n_out = n_out; sc->n_paths = n_paths; sc->n_species = n_species; sc->C = C; sc->in_dim = in_dim; sc->out_dim = out_dim;
    sc->nnz = (int)terms.size();
    // CSR by output row
    std::vector<int> fptr(out_dim + 1, 0), fa1, fa2, fp; std::vector<float> fc;
    for (int R = 0; R < out_dim; ++R) {
        for (const Term &t : terms) if (t.grow == R) { fa1.push_back(t.a1); fa2.push_back(t.a2); fp.push_back(t.p); fc.push_back(t.c); }
        fptr[R + 1] = (int)fa1.size();
    }
    // CSR by input row: a quadratic term contributes to the gradient of both of its factors
    std::vector<int> bptr(in_dim + 1, 0), bo, bg, bp; std::vector<float> bc;
    for (int R = 0; R < in_dim; ++R) {
        for (const Term &t : terms) {
            if (t.a1 == R) { bo.push_back(t.a2); bg.push_back(t.grow); bp.push_back(t.p); bc.push_back(t.c); }
            if (t.a2 == R) { bo.push_back(t.a1); bg.push_back(t.grow); bp.push_back(t.p); bc.push_back(t.c); }
        }
        bptr[R + 1] = (int)bo.size();
    }
    // CSR by path
    std::vector<int> wptr(n_paths + 1, 0), wa1, wa2, wg; std::vector<float> wc;
    for (int p = 0; p < n_paths; ++p) {
        for (const Term &t : terms) if (t.p == p) { wa1.push_back(t.a1); wa2.push_back(t.a2); wg.push_back(t.grow); wc.push_back(t.c); }
        wptr[p + 1] = (int)wa1.size();
    }
    int rc = E3_OK;
    if (device) rc = upload(&sc->f_ptr, fptr);
    if (device && rc == E3_OK) rc = upload(&sc->f_a1, fa1);
    if (device && rc == E3_OK) rc = upload(&sc->f_a2, fa2);
    if (device && rc == E3_OK) rc = upload(&sc->f_p, fp);
    if (device && rc == E3_OK) rc = upload(&sc->f_c, fc);
    if (device && rc == E3_OK) rc = upload(&sc->b_ptr, bptr);
    if (device && rc == E3_OK) rc = upload(&sc->b_other, bo);
    if (device && rc == E3_OK) rc = upload(&sc->b_g, bg);
    if (device && rc == E3_OK) rc = upload(&sc->b_p, bp);
    if (device && rc == E3_OK) rc = upload(&sc->b_c, bc);
    if (device && rc == E3_OK) rc = upload(&sc->w_ptr, wptr);
    if (device && rc == E3_OK) rc = upload(&sc->w_a1, wa1);
    if (device && rc == E3_OK) rc = upload(&sc->w_a2, wa2);
    if (device && rc == E3_OK) rc = upload(&sc->w_g, wg);
    if (device && rc == E3_OK) rc = upload(&sc->w_c, wc);
    // specialised kernels: one NVRTC compilation holds all three (E3_SYMCON_JIT=0 keeps the table-driven ones)
    const char *je = getenv("E3_SYMCON_JIT");
    if (rc == E3_OK && !(je && je[0] == '0') && terms.size() <= 6000) {
        std::vector<ScTerm> ts;
        for (const Term &t : terms) ts.push_back({ t.a1, t.a2, t.grow, t.p, t.c });
        sc->jfwd.name = "e3_sc_fwd";
        sc->jfwd.source = gen_symcon_source(ts, in_dim, out_dim, n_paths);
        sc->jfwd.threads = 128;
        rc = jit_compile(sc->jfwd, "");
        if (rc == E3_OK) {
            sc->jbf = sc->jfwd; sc->jbf.name = "e3_sc_bwd_feats"; sc->jbf.lib = nullptr; sc->jbf.fn = nullptr;
            sc->jbw = sc->jfwd; sc->jbw.name = "e3_sc_bwd_w"; sc->jbw.lib = nullptr; sc->jbw.fn = nullptr;
            sc->jbb = sc->jfwd; sc->jbb.name = "e3_sc_bwd_both"; sc->jbb.lib = nullptr; sc->jbb.fn = nullptr;
            if (regs) *regs = sc->jfwd.regs;
            if (spill) *spill = sc->jfwd.spill;
            if (device) rc = jit_load(sc->jfwd);
            if (device && rc == E3_OK) rc = jit_load(sc->jbf);
            if (device && rc == E3_OK) rc = jit_load(sc->jbw);
            if (device && rc == E3_OK) rc = jit_load(sc->jbb);
            if (device && rc == E3_OK) {        // shared accumulators of the node-chunk kernels: [n_species * n_paths][128] floats
                const long long need = (long long)n_species * n_paths * 128 * (long long)sizeof(float);
                if (need <= 200 * 1024) {
                    sc->acc_smem = (int)need;
                    if (need > 48 * 1024) {
                        cudaError_t e = cudaFuncSetAttribute((const void *)sc->jbw.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)need);
                        if (e == cudaSuccess) e = cudaFuncSetAttribute((const void *)sc->jbb.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)need);
                        if (e != cudaSuccess) rc = cuda_fail(e, "cudaFuncSetAttribute(symmetric contraction accumulators)");
                    }
                    int dev = 0, nsm = 0, occ = 0;
                    cudaGetDevice(&dev);
                    if (rc == E3_OK && cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess &&
                        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, (const void *)sc->jbb.fn, 128, (size_t)need) == cudaSuccess && nsm > 0 && occ > 0)
                        sc->slots = nsm * occ;
                    cudaGetLastError();
                }
            }
            sc->jit = device && rc == E3_OK;
        }
    }
    if (rc != E3_OK || !device) { e3_symcon_destroy(sc); return rc; }
    *out = sc;
    return E3_OK;
}

extern "C" int e3_symcon_create(e3_symcon **out, const e3_irrep *irreps_in, int n_in, const e3_irrep *irreps_out, int n_out, const e3_pair_path *paths,
                                int n_paths, int n_species)
{
    return symcon_create_impl(out, irreps_in, n_in, irreps_out, n_out, paths, n_paths, n_species, true, nullptr, nullptr);
}

extern "C" int e3_symcon_jit_check(const e3_irrep *irreps_in, int n_in, const e3_irrep *irreps_out, int n_out, const e3_pair_path *paths, int n_paths,
                                   int *fwd_regs, int *fwd_spill)
{
    e3_symcon *tmp = nullptr;
    return symcon_create_impl(&tmp, irreps_in, n_in, irreps_out, n_out, paths, n_paths, 1, false, fwd_regs, fwd_spill);
}

extern "C" int e3_symcon_dims(const e3_symcon *sc, int *in_dim, int *out_dim, int *n_paths, int *n_terms)
{
    if (!sc) { set_error("symcon is NULL"); return E3_ERR_INVALID_ARG; }
    if (in_dim) *in_dim = sc->in_dim;
    if (out_dim) *out_dim = sc->out_dim;
    if (n_paths) *n_paths = sc->n_paths;
    if (n_terms) *n_terms = sc->nnz;
    return E3_OK;
}

static inline int block_threads(int C) { return C >= 128 ? 128 : ((C + 31) / 32) * 32; }

extern "C" int e3_symcon_fwd(const e3_symcon *sc, const float *feats, const int32_t *species, const float *weights, int32_t n_nodes, float *out, e3_stream stream)
{
    if (!sc || n_nodes < 0 || (n_nodes > 0 && (!feats || !species || !weights || !out))) { set_error("e3_symcon_fwd: bad arguments"); return E3_ERR_INVALID_ARG; }
    if (n_nodes == 0) return E3_OK;
    if (sc->jit) {
        long long NC = (long long)n_nodes * sc->C;
        int C = sc->C, ns = sc->n_species;
        void *args[] = { (void *)&feats, (void *)&species, (void *)&weights, (void *)&NC, (void *)&C, (void *)&ns, (void *)&out };
        E3_CUDA_TRY(cudaLaunchKernel((const void *)sc->jfwd.fn, dim3((unsigned)((NC + 127) / 128)), dim3(128), args, 0, reinterpret_cast<cudaStream_t>(stream)));
        return E3_OK;
    }
    const int th = block_threads(sc->C);
    const size_t smem = (size_t)sc->in_dim * th * sizeof(float);
    symcon_fwd_kernel<<<dim3((unsigned)n_nodes, (unsigned)((sc->C + th - 1) / th)), th, smem, reinterpret_cast<cudaStream_t>(stream)>>>(
        feats, species, weights, sc->C, sc->in_dim, sc->out_dim, sc->n_paths, sc->n_species, sc->f_ptr, sc->f_a1, sc->f_a2, sc->f_p, sc->f_c, out);
    E3_CUDA_TRY(cudaGetLastError());
    return E3_OK;
}

extern "C" size_t e3_symcon_workspace_bytes(const e3_symcon *sc, int32_t n_nodes)
{
    if (!sc) return 0;
    const long long per = (long long)sc->n_species * sc->n_paths * sc->C;
    return (size_t)symcon_chunks(n_nodes, sc->C, per, sc->slots) * per * sizeof(float) + 256;
}

extern "C" int e3_symcon_bwd(const e3_symcon *sc, const float *feats, const int32_t *species, const float *weights, int32_t n_nodes, const float *grad_out,
                             float *grad_feats, float *grad_weights, void *workspace, size_t workspace_bytes, e3_stream stream)
{
    if (!sc || n_nodes < 0 || (n_nodes > 0 && (!feats || !species || !weights || !grad_out))) { set_error("e3_symcon_bwd: bad arguments"); return E3_ERR_INVALID_ARG; }
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    if (sc->jit) {
        long long NC = (long long)n_nodes * sc->C;
        int C = sc->C, ns = sc->n_species, N = n_nodes;
        const int total = sc->n_species * sc->n_paths * sc->C;
        int chunks = symcon_chunks(n_nodes, sc->C, total, sc->slots);
        float *partial = reinterpret_cast<float *>(workspace);
        if (grad_weights && (!workspace || workspace_bytes < e3_symcon_workspace_bytes(sc, n_nodes))) { set_error("e3_symcon_bwd: workspace too small"); return E3_ERR_WORKSPACE; }
        const bool chunk_kernels = grad_weights && sc->acc_smem > 0 && n_nodes > 0;
        if (grad_feats && n_nodes > 0 && !chunk_kernels) {
            void *args[] = { (void *)&feats, (void *)&species, (void *)&weights, (void *)&grad_out, (void *)&NC, (void *)&C, (void *)&ns, (void *)&grad_feats };
            E3_CUDA_TRY(cudaLaunchKernel((const void *)sc->jbf.fn, dim3((unsigned)((NC + 127) / 128)), dim3(128), args, 0, st));
        }
        if (chunk_kernels) {           // one pass over feats and grad_out for both gradients (or for grad_weights alone)
            void *args[] = { (void *)&feats, (void *)&species, (void *)&weights, (void *)&grad_out, (void *)&N, (void *)&C, (void *)&ns, (void *)&chunks,
                             (void *)&grad_feats, (void *)&partial };
            const cudaKernel_t fn = grad_feats ? sc->jbb.fn : sc->jbw.fn;
            E3_CUDA_TRY(cudaLaunchKernel((const void *)fn, dim3((unsigned)(((long long)chunks * C + 127) / 128)), dim3(128), args, (size_t)sc->acc_smem, st));
        } else if (grad_weights) {     // accumulators too large for shared memory (or no nodes): table-driven partial sums
            const int pc = sc->n_paths * sc->C;
            symcon_bwd_w_partial_kernel<<<dim3((unsigned)chunks, (unsigned)((pc + 127) / 128)), 128, 0, st>>>(
                feats, species, grad_out, sc->C, sc->in_dim, sc->out_dim, sc->n_paths, sc->n_species, n_nodes, chunks, sc->w_ptr, sc->w_a1, sc->w_a2, sc->w_g, sc->w_c, partial);
            E3_CUDA_TRY(cudaGetLastError());
        }
        if (grad_weights) {
            symcon_bwd_w_reduce_kernel<<<(unsigned)((total + 31) / 32), dim3(32, 32), 0, st>>>(partial, total, chunks, grad_weights);
            E3_CUDA_TRY(cudaGetLastError());
        }
        return E3_OK;
    }
    const int th = block_threads(sc->C);
    if (grad_feats && n_nodes > 0) {
        const size_t smem = (size_t)(sc->in_dim + sc->out_dim) * th * sizeof(float);
        if (smem > 48 * 1024) {
            static bool set = false;
            if (!set) { E3_CUDA_TRY(cudaFuncSetAttribute(symcon_bwd_feats_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024)); set = true; }
            if (smem > 200 * 1024) { set_error("e3_symcon_bwd: rows too long for shared memory"); return E3_ERR_UNSUPPORTED; }
        }
        symcon_bwd_feats_kernel<<<dim3((unsigned)n_nodes, (unsigned)((sc->C + th - 1) / th)), th, smem, st>>>(
            feats, species, weights, grad_out, sc->C, sc->in_dim, sc->out_dim, sc->n_paths, sc->n_species, sc->b_ptr, sc->b_other, sc->b_g, sc->b_p, sc->b_c, grad_feats);
        E3_CUDA_TRY(cudaGetLastError());
    }
    if (grad_weights) {
        if (!workspace || workspace_bytes < e3_symcon_workspace_bytes(sc, n_nodes)) { set_error("e3_symcon_bwd: workspace too small"); return E3_ERR_WORKSPACE; }
        float *partial = reinterpret_cast<float *>(workspace);
        const int pc = sc->n_paths * sc->C, total = sc->n_species * pc, chunks = symcon_chunks(n_nodes, sc->C, total, sc->slots);
        symcon_bwd_w_partial_kernel<<<dim3((unsigned)chunks, (unsigned)((pc + 127) / 128)), 128, 0, st>>>(
            feats, species, grad_out, sc->C, sc->in_dim, sc->out_dim, sc->n_paths, sc->n_species, n_nodes, chunks, sc->w_ptr, sc->w_a1, sc->w_a2, sc->w_g, sc->w_c, partial);
        E3_CUDA_TRY(cudaGetLastError());
        symcon_bwd_w_reduce_kernel<<<(unsigned)((total + 31) / 32), dim3(32, 32), 0, st>>>(partial, total, chunks, grad_weights);
        E3_CUDA_TRY(cudaGetLastError());
    }
    return E3_OK;
}
