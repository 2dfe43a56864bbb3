// C ABI entry points (include/e3b200.h): argument checking, launches, the host-buffer session.
#include <algorithm>
#include <cstdio>
#include <cstring>
#include <new>

#include "e3_internal.h"

using namespace e3;

static inline cudaStream_t S(e3_stream s) { return reinterpret_cast<cudaStream_t>(s); }
static inline bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
static inline size_t esize(const e3_plan *pl) { return pl->dtype == E3_BF16 ? 2 : 4; }

extern "C" const char *e3_status_string(int status)
{
    switch (status) {
    case E3_OK: return "ok";
    case E3_ERR_INVALID_ARG: return "invalid argument";
    case E3_ERR_BAD_PATH: return "path violates triangle/parity/index rule";
    case E3_ERR_UNSUPPORTED: return "unsupported configuration";
    case E3_ERR_UNSORTED: return "receivers not sorted";
    case E3_ERR_CUDA: return "CUDA error or no device";
    case E3_ERR_JIT: return "kernel specialisation failed";
    case E3_ERR_WORKSPACE: return "workspace missing or too small";
    default: return "unknown status";
    }
}

extern "C" const char *e3_last_error(void) { return get_error(); }

// dynamic shared memory of the third-generation forward when `f` sub-teams share a receiver
static int v3_smem(const e3_plan *pl, int f)
{
    const int ring = f * pl->fwd_v3_depth * pl->fwd_v3_stage, part = (f - 1) * pl->fwd_v3_part;
    return pl->fwd_v3_bar + (ring > part ? ring : part);
}
static int v3_fsplit_max(const e3_plan *pl)
{
    int f = 4;
    while (f > 1 && (v3_smem(pl, f) > 227 * 1024 || pl->fwd_tw * 32 * f > 1024)) f >>= 1;
    return f;
}

// ---------------------------------------------------------------------------------------------
// plan
// ---------------------------------------------------------------------------------------------
static int plan_generate(e3_plan &pl, const char *src_path)
{
    plan_make_roles(pl);
    pl.fwd.name = "e3_fwd";
    pl.bwd.name = "e3_bwd";
    pl.fwd.source = pl.fwd_v3 ? gen_forward_v3(pl) : (pl.v2 ? gen_forward_v2(pl) : gen_forward_source(pl));
    pl.bwd.source = pl.bwd_v2 ? gen_backward_v2(pl) : gen_backward_source(pl);
    pl.fwd.threads = pl.fwd_v3 ? pl.fwd_tw * 32 : pl.fwd_warps * 32;
    pl.bwd.threads = pl.bwd_warps * 32;
    std::string f1, f2;
    if (src_path) { f1 = std::string(src_path) + ".fwd.cu"; f2 = std::string(src_path) + ".bwd.cu"; }
    int rc = jit_compile(pl.fwd, f1);
    if (rc != E3_OK) return rc;
    return jit_compile(pl.bwd, f2);
}

// generate + compile + load the two kernels of a regular plan (or of one sub-plan of a composite)
static int plan_finish(e3_plan *pl)
{
    int rc = plan_generate(*pl, nullptr);
    if (rc == E3_OK) rc = jit_load(pl->fwd);
    if (rc == E3_OK) rc = jit_load(pl->bwd);
    const int fwd_smem_max = (rc == E3_OK && pl->fwd_v3) ? v3_smem(pl, v3_fsplit_max(pl)) : pl->fwd.smem_dyn;
    if (rc == E3_OK && fwd_smem_max > 48 * 1024 &&
        cudaFuncSetAttribute((const void *)pl->fwd.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, fwd_smem_max) != cudaSuccess)
        rc = cuda_fail(cudaGetLastError(), "cudaFuncSetAttribute(fwd smem)");
    if (rc == E3_OK && pl->fwd_v3) {       // zeros: the operands of the missing edges of a receiver's last step
        pl->zeros_bytes = (size_t)std::max(pl->in_dim, (int)pl->paths.size()) * pl->C * 4 + 256;
        cudaError_t e = cudaMalloc(&pl->zeros, pl->zeros_bytes);
        if (e == cudaSuccess) e = cudaMemset(pl->zeros, 0, pl->zeros_bytes);
        if (e != cudaSuccess) rc = cuda_fail(e, "plan zeros buffer");
    }
    if (rc == E3_OK && pl->bwd.smem_dyn > 48 * 1024 &&
        cudaFuncSetAttribute((const void *)pl->bwd.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, pl->bwd.smem_dyn) != cudaSuccess)
        rc = cuda_fail(cudaGetLastError(), "cudaFuncSetAttribute(bwd smem)");
    if (rc == E3_OK) {
        int dev = 0, nsm = 0, a = 0, b = 0;
        cudaGetDevice(&dev);
        if (cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && nsm > 0) pl->n_sm = nsm;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&a, (const void *)pl->fwd.fn, pl->fwd.threads, pl->fwd.smem_dyn) == cudaSuccess && a > 0) pl->fwd_ctas_per_sm = a;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, (const void *)pl->bwd.fn, pl->bwd.threads, pl->bwd.smem_dyn) == cudaSuccess && b > 0) pl->bwd_ctas_per_sm = b;
        cudaGetLastError();
    }
    return rc;
}

static void plan_free(e3_plan *pl)
{
    if (!pl) return;
    for (e3_plan *sp : pl->subs) plan_free(sp);
    for (cudaEvent_t ev : pl->ov_ev) if (ev) cudaEventDestroy(ev);
    if (pl->side_stream) cudaStreamDestroy(pl->side_stream);
    jit_unload(pl->fwd);
    jit_unload(pl->bwd);
    if (pl->zeros) cudaFree(pl->zeros);
    delete pl;
}

extern "C" int e3_plan_create(e3_plan **plan, const e3_irrep *irreps_in, int n_in, int sh_lmax, const e3_irrep *irreps_out,
                              int n_out, const e3_path *paths, int n_paths, e3_dtype dtype)
{
    if (!plan) { set_error("e3_plan_create: plan is NULL"); return E3_ERR_INVALID_ARG; }
    *plan = nullptr;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        set_error("e3_plan_create: no CUDA device (this library has no CPU fallback)");
        return E3_ERR_CUDA;
    }
    e3_plan *pl = new (std::nothrow) e3_plan();
    if (!pl) { set_error("out of host memory"); return E3_ERR_INVALID_ARG; }
    int rc;
    if (plan_is_composite(irreps_in, n_in, irreps_out, n_out)) {
        // NEXT-4: per-irrep multiplicities -> one generated sub-plan per multiplicity class
        rc = plan_build_composite(*pl, irreps_in, n_in, sh_lmax, irreps_out, n_out, paths, n_paths, dtype, /*cg_on_device=*/true);
        for (size_t k = 0; rc == E3_OK && k < pl->subs.size(); ++k) rc = plan_finish(pl->subs[k]);
    } else {
        rc = plan_build_tables(*pl, irreps_in, n_in, sh_lmax, irreps_out, n_out, paths, n_paths, dtype, /*cg_on_device=*/true);
        if (rc == E3_OK) rc = plan_finish(pl);
    }
    if (rc == E3_OK) {       // side stream + events of the VJP overlap
        cudaError_t e = cudaStreamCreateWithFlags(&pl->side_stream, cudaStreamNonBlocking);
        for (int k = 0; k <= e3_plan::kMaxOverlap && e == cudaSuccess; ++k) e = cudaEventCreateWithFlags(&pl->ov_ev[k], cudaEventDisableTiming);
        if (e != cudaSuccess) rc = cuda_fail(e, "plan side stream");
    }
    if (rc != E3_OK) { plan_free(pl); return rc; }
    *plan = pl;
    return E3_OK;
}

extern "C" int e3_plan_destroy(e3_plan *plan)
{
    plan_free(plan);
    return E3_OK;
}

extern "C" int e3_plan_sizes(const e3_plan *plan, int64_t *feats_per_node, int64_t *out_per_node, int64_t *weights_per_edge)
{
    if (!plan) { set_error("plan is NULL"); return E3_ERR_INVALID_ARG; }
    if (feats_per_node) *feats_per_node = plan->in_size();
    if (out_per_node) *out_per_node = plan->out_size();
    if (weights_per_edge) *weights_per_edge = plan->w_size();
    return E3_OK;
}

extern "C" int e3_plan_dims(const e3_plan *plan, int *in_dim, int *sh_dim, int *out_dim, int *weights_per_edge, int *nnz_total)
{
    if (!plan) { set_error("plan is NULL"); return E3_ERR_INVALID_ARG; }
    if (in_dim) *in_dim = plan->in_dim;
    if (sh_dim) *sh_dim = plan->sh_dim;
    if (out_dim) *out_dim = plan->out_dim;
    if (weights_per_edge) *weights_per_edge = plan->w_size();
    if (nnz_total) *nnz_total = plan->nnz_total;
    return E3_OK;
}

extern "C" int e3_plan_get_cg(const e3_plan *plan, int path, int *m1, int *m2, int *m3, double *coef, int *nnz)
{
    if (!plan || !nnz || path < 0 || path >= (int)plan->paths.size()) { set_error("e3_plan_get_cg: bad arguments"); return E3_ERR_INVALID_ARG; }
    if (!plan->subs.empty()) return e3_plan_get_cg(plan->subs[plan->path_map[path].first], plan->path_map[path].second, m1, m2, m3, coef, nnz);
    const PathInfo &pi = plan->paths[path];
    *nnz = (int)pi.nz.size();
    if (m1 && m2 && m3 && coef)
        for (size_t i = 0; i < pi.nz.size(); ++i) { m1[i] = pi.nz[i].m1; m2[i] = pi.nz[i].m2; m3[i] = pi.nz[i].m3; coef[i] = pi.nz[i].c; }
    return E3_OK;
}

extern "C" int e3_plan_kernel_info(const e3_plan *plan, int which, int *regs, int *spill_bytes, int *smem_bytes,
                                   int *threads_per_block, int *n_roles, int *channels_per_lane)
{
    if (!plan || (which != 0 && which != 1)) { set_error("e3_plan_kernel_info: bad arguments"); return E3_ERR_INVALID_ARG; }
    if (!plan->subs.empty()) {
        int a[6] = { 0, 0, 0, 0, 0, 0 };
        for (const e3_plan *sp : plan->subs) {
            int b[6];
            e3_plan_kernel_info(sp, which, &b[0], &b[1], &b[2], &b[3], &b[4], &b[5]);
            for (int i = 0; i < 6; ++i) a[i] = i == 4 ? a[i] + b[i] : std::max(a[i], b[i]);
        }
        if (regs) *regs = a[0];
        if (spill_bytes) *spill_bytes = a[1];
        if (smem_bytes) *smem_bytes = a[2];
        if (threads_per_block) *threads_per_block = a[3];
        if (n_roles) *n_roles = a[4];
        if (channels_per_lane) *channels_per_lane = a[5];
        return E3_OK;
    }
    const JitKernel &k = which == 0 ? plan->fwd : plan->bwd;
    if (regs) *regs = k.regs;
    if (spill_bytes) *spill_bytes = k.spill;
    if (smem_bytes) *smem_bytes = k.smem + k.smem_dyn;
    if (threads_per_block) *threads_per_block = k.threads;
    if (n_roles) *n_roles = which == 0 ? (int)plan->roles.size() : (plan->bwd_v2 ? plan->bwd_nroles : 1);
    if (channels_per_lane) *channels_per_lane = ((which == 0 && plan->v2) || (which == 1 && plan->bwd_v2)) ? 4 : plan->K;
    return E3_OK;
}

extern "C" int e3_plan_work(const e3_plan *plan, double *fwd_flop_per_edge, double *bwd_flop_per_edge)
{
    if (!plan) { set_error("plan is NULL"); return E3_ERR_INVALID_ARG; }
    double f = 0, b = 0;
    for (const e3_plan *sp : plan->subs) {
        double f1 = 0, b1 = 0;
        e3_plan_work(sp, &f1, &b1);
        f += f1; b += b1;
    }
    if (plan->subs.empty())
    for (const PathInfo &pi : plan->paths) {
        f += plan->C * (2.0 * pi.nzM + 2.0 * (2 * pi.l3 + 1)) + 2.0 * pi.nz.size();
        b += plan->C * (6.0 * pi.nzM + 3.0 * (2 * pi.l3 + 1)) + 4.0 * pi.nz.size();
    }
    if (fwd_flop_per_edge) *fwd_flop_per_edge = f;
    if (bwd_flop_per_edge) *bwd_flop_per_edge = b;
    return E3_OK;
}

extern "C" int e3_jit_check(const e3_irrep *irreps_in, int n_in, int sh_lmax, const e3_irrep *irreps_out, int n_out,
                            const e3_path *paths, int n_paths, e3_dtype dtype, const char *src_path, int *fwd_regs,
                            int *fwd_spill, int *bwd_regs, int *bwd_spill)
{
    e3_plan pl;
    if (plan_is_composite(irreps_in, n_in, irreps_out, n_out)) {
        int rc = plan_build_composite(pl, irreps_in, n_in, sh_lmax, irreps_out, n_out, paths, n_paths, dtype, /*cg_on_device=*/false);
        int v[4] = { 0, 0, 0, 0 };
        for (size_t k = 0; rc == E3_OK && k < pl.subs.size(); ++k) {
            const std::string sp = src_path ? std::string(src_path) + ".class" + std::to_string(k) : std::string();
            rc = plan_generate(*pl.subs[k], src_path ? sp.c_str() : nullptr);
            v[0] = std::max(v[0], pl.subs[k]->fwd.regs); v[1] = std::max(v[1], pl.subs[k]->fwd.spill);
            v[2] = std::max(v[2], pl.subs[k]->bwd.regs); v[3] = std::max(v[3], pl.subs[k]->bwd.spill);
        }
        for (e3_plan *sp : pl.subs) delete sp;
        pl.subs.clear();
        if (rc != E3_OK) return rc;
        if (fwd_regs) *fwd_regs = v[0];
        if (fwd_spill) *fwd_spill = v[1];
        if (bwd_regs) *bwd_regs = v[2];
        if (bwd_spill) *bwd_spill = v[3];
        return E3_OK;
    }
    int rc = plan_build_tables(pl, irreps_in, n_in, sh_lmax, irreps_out, n_out, paths, n_paths, dtype, /*cg_on_device=*/false);
    if (rc == E3_OK) rc = plan_generate(pl, src_path);
    if (rc != E3_OK) return rc;
    if (fwd_regs) *fwd_regs = pl.fwd.regs;
    if (fwd_spill) *fwd_spill = pl.fwd.spill;
    if (bwd_regs) *bwd_regs = pl.bwd.regs;
    if (bwd_spill) *bwd_spill = pl.bwd.spill;
    return E3_OK;
}

// ---------------------------------------------------------------------------------------------
// graph, SH, forces
// ---------------------------------------------------------------------------------------------
extern "C" size_t e3_graph_workspace_bytes(int64_t n_edges, int32_t n_nodes)
{
    if (n_edges < 0 || n_nodes < 0) return 0;
    return graph_workspace_bytes(n_edges, n_nodes);
}

extern "C" int e3_graph_prepare(const int32_t *senders, const int32_t *receivers, int64_t n_edges, int32_t n_nodes,
                                int32_t *row_ptr, int32_t *perm_s, int32_t *col_ptr, void *workspace, size_t workspace_bytes,
                                int validate, e3_stream stream)
{
    if (n_edges < 0 || n_nodes < 0 || n_edges > 0x7fffffffLL || !row_ptr || !col_ptr || (n_edges > 0 && (!senders || !receivers || !perm_s))) {
        set_error("e3_graph_prepare: bad arguments");
        return E3_ERR_INVALID_ARG;
    }
    return launch_graph_prepare(senders, receivers, n_edges, n_nodes, row_ptr, perm_s, col_ptr, workspace, workspace_bytes, validate, S(stream));
}

extern "C" int e3_sh_fwd(const e3_plan *plan, const float *vec, int64_t n_edges, void *sh, e3_stream stream)
{
    if (!plan || n_edges < 0 || (n_edges > 0 && (!vec || !sh))) { set_error("e3_sh_fwd: bad arguments"); return E3_ERR_INVALID_ARG; }
    return launch_sh_fwd(plan->sh_lmax, plan->dtype, vec, n_edges, sh, S(stream));
}

extern "C" int e3_sh_bwd(const e3_plan *plan, const float *vec, const float *grad_sh, int64_t n_edges, float *grad_vec, e3_stream stream)
{
    if (!plan || n_edges < 0 || (n_edges > 0 && (!vec || !grad_sh || !grad_vec))) { set_error("e3_sh_bwd: bad arguments"); return E3_ERR_INVALID_ARG; }
    return launch_sh_bwd(plan->sh_lmax, vec, grad_sh, n_edges, grad_vec, S(stream));
}

extern "C" int e3_force_reduce(const float *grad_vec, const int32_t *row_ptr, const int32_t *perm_s, const int32_t *col_ptr,
                               int64_t n_edges, int32_t n_nodes, float *forces, e3_stream stream)
{
    if (n_edges < 0 || n_nodes < 0 || !row_ptr || !col_ptr || (n_nodes > 0 && !forces) || (n_edges > 0 && (!grad_vec || !perm_s))) {
        set_error("e3_force_reduce: bad arguments");
        return E3_ERR_INVALID_ARG;
    }
    return launch_force_reduce(grad_vec, row_ptr, perm_s, col_ptr, n_edges, n_nodes, forces, S(stream));
}

// ---------------------------------------------------------------------------------------------
// tensor product + scatter
// ---------------------------------------------------------------------------------------------
// launches the forward kernel for the receivers whose row_ptr / out rows start at the given pointers (a receiver range
// of a larger graph is the same call with offset pointers: edge-indexed and sender-indexed tensors stay absolute)
static int launch_fwd(const e3_plan *plan, const void *feats, const void *sh, const void *weights, const int32_t *senders,
                      const int32_t *row_ptr, int32_t n_nodes, float *out, cudaStream_t st, int32_t heur_nodes = -1)
{
    if (heur_nodes < 0) heur_nodes = n_nodes;     // launch-shape heuristics follow the size of the WHOLE graph
    if (n_nodes == 0) return E3_OK;
    if (!plan->subs.empty()) {                    // composite: every multiplicity class writes its own output blocks
        for (const e3_plan *sp : plan->subs) {
            const int rc = launch_fwd(sp, feats, sh, weights, senders, row_ptr, n_nodes, out, st, heur_nodes);
            if (rc != E3_OK) return rc;
        }
        return E3_OK;
    }
    if (!plan->fwd.fn) { set_error("plan has no loaded forward kernel"); return E3_ERR_CUDA; }
    // small graphs (v2 kernels): `fsplit` warps share one (receiver, role) so that the grid covers the machine
    // several times over; the result depends on fsplit only through the (fixed) summation grouping
    int fsplit = 1;
    const long long nchb = plan->v2 ? plan->nchb2 : plan->nchb;
    if (plan->fwd_v3) {
        // one CTA per (receiver, team, channel block); small graphs: `fsplit` sub-teams share a receiver (each takes a
        // contiguous run of its edge steps, partial sums added in sub-team order), so that the grid still covers the
        // machine several times over
        const long long nteams = (long long)plan->teams.size();
        fsplit = plan->fwd_split;
        if (fsplit <= 0) {
            const double waves = (double)heur_nodes * nteams * nchb / ((double)plan->n_sm * plan->fwd_ctas_per_sm);
            fsplit = waves >= 6.0 ? 1 : (waves >= 3.0 ? 2 : 4);
        }
        if (fsplit != 1 && fsplit != 2 && fsplit != 4) fsplit = 1;
        const int fmax = v3_fsplit_max(plan);
        if (fsplit > fmax) fsplit = fmax;
        const long long chunk_sz = plan->fwd_v3_chunk < n_nodes ? plan->fwd_v3_chunk : n_nodes;
        const long long chunks = ((long long)n_nodes + chunk_sz - 1) / chunk_sz;
        const long long grid3 = chunks * chunk_sz * nteams * nchb;
        if (grid3 > 0x7fffffffLL) { set_error("grid too large"); return E3_ERR_UNSUPPORTED; }
        const void *zeros = plan->zeros;
        int chunk_i = (int)chunk_sz;
        void *args3[] = { (void *)&feats, (void *)&sh, (void *)&weights, (void *)&senders, (void *)&row_ptr, (void *)&out, (void *)&n_nodes, (void *)&fsplit, (void *)&zeros, (void *)&chunk_i };
        E3_CUDA_TRY(cudaLaunchKernel((const void *)plan->fwd.fn, dim3((unsigned)grid3), dim3(plan->fwd_tw * 32 * fsplit), args3, v3_smem(plan, fsplit), st));
        return E3_OK;
    }
    if (plan->v2) {
        fsplit = plan->fwd_split;
        if (fsplit <= 0) {
            const double waves = (double)heur_nodes * plan->roles.size() * nchb /
                                 ((double)plan->n_sm * plan->fwd_ctas_per_sm * plan->fwd_warps);
            fsplit = waves >= 6.0 ? 1 : (waves >= 3.0 ? 2 : 4);
        }
        if (fsplit != 1 && fsplit != 2 && fsplit != 4) fsplit = 1;
        while (plan->fwd_warps % fsplit) fsplit >>= 1;
    }
    const long long per_chunk = (long long)plan->fwd_chunk * (plan->fwd_warps / fsplit);     // receivers per chunk
    const long long chunks = (n_nodes + per_chunk - 1) / per_chunk;
    long long grid = chunks * plan->fwd_chunk * (long long)plan->roles.size() * nchb;
    if (grid > 0x7fffffffLL) { set_error("grid too large"); return E3_ERR_UNSUPPORTED; }
    void *args[] = { (void *)&feats, (void *)&sh, (void *)&weights, (void *)&senders, (void *)&row_ptr, (void *)&out, (void *)&n_nodes, (void *)&fsplit };
    E3_CUDA_TRY(cudaLaunchKernel((const void *)plan->fwd.fn, dim3((unsigned)grid), dim3(plan->fwd.threads), args, plan->fwd.smem_dyn, st));
    return E3_OK;
}

extern "C" int e3_tp_scatter_fwd(const e3_plan *plan, const void *feats, const void *sh, const void *weights,
                                 const int32_t *senders, const int32_t *receivers, const int32_t *row_ptr, int64_t n_edges,
                                 int32_t n_nodes, float *out, e3_stream stream)
{
    (void)receivers;
    if (!plan || n_edges < 0 || n_nodes < 0 || !row_ptr || (n_nodes > 0 && (!feats || !out)) ||
        (n_edges > 0 && (!sh || !weights || !senders))) {
        set_error("e3_tp_scatter_fwd: bad arguments");
        return E3_ERR_INVALID_ARG;
    }
    if (!aligned16(feats) || !aligned16(weights) || !aligned16(out) || !aligned16(sh)) {
        set_error("e3_tp_scatter_fwd: tensor pointers must be 16-byte aligned");
        return E3_ERR_INVALID_ARG;
    }
    return launch_fwd(plan, feats, sh, weights, senders, row_ptr, n_nodes, out, S(stream));
}

// partial grad_sh buffers of the VJP: one per backward role, for a composite one per (class, role); 0 = written in place
static int gsh_parts(const e3_plan *plan)
{
    if (!plan->subs.empty()) {
        int n = 0;
        for (const e3_plan *sp : plan->subs) n += sp->bwd_v2 ? sp->bwd_nroles : 1;
        return n;
    }
    return (plan->bwd_v2 && plan->bwd_nroles > 1) ? plan->bwd_nroles : 0;
}

extern "C" size_t e3_bwd_workspace_bytes(const e3_plan *plan, int64_t n_edges, int32_t n_nodes)
{
    (void)n_nodes;
    if (!plan || n_edges < 0) return 0;
    size_t b = (((size_t)n_edges * plan->in_size() * sizeof(float) + 255) / 256) * 256 + 256;     // per-edge grad_feats rows
    b += (size_t)gsh_parts(plan) * n_edges * plan->sh_dim * sizeof(float) + 256;   // per-role (and per-class) grad_sh
    return b;
}

static size_t gsh_parts_offset(const e3_plan *plan, int64_t n_edges)
{
    return (((size_t)n_edges * plan->in_size() * sizeof(float) + 255) / 256) * 256;
}

// first VJP phase for a receiver range (offset row_ptr / grad_out pointers, absolute edge- and sender-indexed tensors):
// grad_weights, per-edge grad_feats rows (workspace) and grad_sh (per-role partial buffers when the plan has several roles)
static int launch_bwd_phase1(const e3_plan *plan, const void *feats, const void *sh, const void *weights, const int32_t *senders,
                             const int32_t *row_ptr, int32_t n_nodes, const float *grad_out, float *grad_sh, void *grad_weights,
                             void *workspace, int64_t n_edges_total, cudaStream_t st, int32_t heur_nodes = -1, float *gsh_part = nullptr)
{
    if (n_nodes == 0 || n_edges_total == 0) return E3_OK;
    if (heur_nodes < 1) heur_nodes = n_nodes;
    if (!plan->subs.empty()) {       // composite: the classes share the per-edge workspace rows; each (class, role) has its grad_sh part
        float *parts = reinterpret_cast<float *>(reinterpret_cast<char *>(workspace) + gsh_parts_offset(plan, n_edges_total));
        for (const e3_plan *sp : plan->subs) {
            const int rc = launch_bwd_phase1(sp, feats, sh, weights, senders, row_ptr, n_nodes, grad_out, grad_sh, grad_weights, workspace,
                                             n_edges_total, st, heur_nodes, parts);
            if (rc != E3_OK) return rc;
            parts += (size_t)(sp->bwd_v2 ? sp->bwd_nroles : 1) * n_edges_total * plan->sh_dim;
        }
        return E3_OK;
    }
    if (!plan->bwd.fn) { set_error("plan has no loaded backward kernel"); return E3_ERR_CUDA; }
    float *dxe = (float *)workspace;
    const int roles = plan->bwd_v2 ? plan->bwd_nroles : 1;
    // one CTA per (receiver, role, part); its warps split the receiver's edges.  Small graphs are cut into `split`
    // parts per receiver so that the grid still covers the machine several times over (tail effect).
    int split = 1;
    if (plan->bwd_v2) {
        split = plan->bwd_split;
        if (split <= 0) {
            const long long slots = (long long)plan->n_sm * plan->bwd_ctas_per_sm;
            split = (int)((8 * slots + heur_nodes - 1) / heur_nodes);
            split = split < 1 ? 1 : (split > 4 ? 4 : split);
        }
    }
    long long grid = (long long)n_nodes * split;
    if (plan->bwd_v2) {           // CTA order: chunk of receivers, then role, then (receiver, part)
        const long long chunks = ((long long)n_nodes + plan->bwd_chunk - 1) / plan->bwd_chunk;
        grid = chunks * plan->bwd_chunk * plan->bwd_nroles * split;
    }
    if (grid > 0x7fffffffLL) { set_error("grid too large"); return E3_ERR_UNSUPPORTED; }
    float *gsh_arg = gsh_part ? gsh_part
                              : (roles > 1 ? reinterpret_cast<float *>(reinterpret_cast<char *>(workspace) + gsh_parts_offset(plan, n_edges_total)) : grad_sh);
    long long ne = n_edges_total;
    void *args[] = { (void *)&feats, (void *)&sh, (void *)&weights, (void *)&senders, (void *)&row_ptr, (void *)&grad_out,
                     (void *)&dxe, (void *)&gsh_arg, (void *)&grad_weights, (void *)&n_nodes, (void *)&split, (void *)&ne };
    E3_CUDA_TRY(cudaLaunchKernel((const void *)plan->bwd.fn, dim3((unsigned)grid), dim3(plan->bwd.threads), args, plan->bwd.smem_dyn, st));
    return E3_OK;
}

// second VJP phase: per-sender sum of the workspace rows, sum of the per-role grad_sh buffers
static int launch_bwd_phase2(const e3_plan *plan, const int32_t *perm_s, const int32_t *col_ptr, int64_t n_edges, int32_t n_nodes,
                             float *grad_feats, float *grad_sh, void *workspace, cudaStream_t st)
{
    const int roles = gsh_parts(plan);
    int rc = launch_dx_reduce((const float *)workspace, perm_s, col_ptr, n_nodes, plan->in_size(), grad_feats, st);
    if (rc == E3_OK && roles > 0 && n_edges > 0)
        rc = launch_gsh_reduce(reinterpret_cast<const float *>(reinterpret_cast<const char *>(workspace) + gsh_parts_offset(plan, n_edges)),
                               roles, n_edges * plan->sh_dim, grad_sh, st);
    return rc;
}

extern "C" int e3_tp_scatter_bwd(const e3_plan *plan, const void *feats, const void *sh, const void *weights,
                                 const int32_t *senders, const int32_t *receivers, const int32_t *row_ptr, const int32_t *perm_s,
                                 const int32_t *col_ptr, int64_t n_edges, int32_t n_nodes, const float *grad_out,
                                 float *grad_feats, float *grad_sh, void *grad_weights, void *workspace, size_t workspace_bytes,
                                 e3_stream stream)
{
    (void)receivers;
    if (!plan || n_edges < 0 || n_nodes < 0 || !col_ptr || !row_ptr || (n_nodes > 0 && (!feats || !grad_out || !grad_feats)) ||
        (n_edges > 0 && (!sh || !weights || !senders || !perm_s || !grad_sh))) {
        set_error("e3_tp_scatter_bwd: bad arguments");
        return E3_ERR_INVALID_ARG;
    }
    if (!aligned16(feats) || !aligned16(weights) || !aligned16(grad_out) || !aligned16(grad_feats) || !aligned16(grad_weights) ||
        !aligned16(sh) || !aligned16(workspace) || !aligned16(grad_sh)) {
        set_error("e3_tp_scatter_bwd: tensor pointers must be 16-byte aligned");
        return E3_ERR_INVALID_ARG;
    }
    if (n_edges > 0 && (!workspace || workspace_bytes < e3_bwd_workspace_bytes(plan, n_edges, n_nodes))) {
        set_error("e3_tp_scatter_bwd: workspace too small (need %zu bytes)", e3_bwd_workspace_bytes(plan, n_edges, n_nodes));
        return E3_ERR_WORKSPACE;
    }
    if (n_nodes == 0) return E3_OK;
    cudaStream_t st = S(stream);
    // opt-in overlap of the two phases (E3_TUNE bwd_overlap=K): K receiver chunks of the first phase on `stream`, the per-sender reduction
    // of the senders each chunk completes on the plan's side stream; the side stream is joined before returning, so the call keeps its
    // single-stream semantics (and can be graph-captured).  Measured on config 4 (power-capped B200): 31.8 ms off, 32.2 / 32.6 / 33.3 ms
    // with 4 / 8 / 16 chunks -- the reduction's energy moves, it does not disappear, and every chunk adds a tail -- so it is OFF by default.
    int chunks = plan->bwd_overlap;
    if (chunks < 0) chunks = 0;
    if (chunks > e3_plan::kMaxOverlap) chunks = e3_plan::kMaxOverlap;
    if (chunks >= 2 && receivers && n_edges > 0 && plan->side_stream) {
        const size_t out_row = (size_t)plan->out_size();
        E3_CUDA_TRY(cudaEventRecord(plan->ov_ev[e3_plan::kMaxOverlap], st));                 // fork: the side stream starts after earlier work of `stream`
        E3_CUDA_TRY(cudaStreamWaitEvent(plan->side_stream, plan->ov_ev[e3_plan::kMaxOverlap], 0));
        int32_t r_lo = 0;
        for (int k = 0; k < chunks; ++k) {
            const int32_t r_hi = k + 1 == chunks ? n_nodes : (int32_t)(((int64_t)n_nodes * (k + 1)) / chunks);
            if (r_hi <= r_lo) continue;
            int rc = launch_bwd_phase1(plan, feats, sh, weights, senders, row_ptr + r_lo, r_hi - r_lo, grad_out + (size_t)r_lo * out_row, grad_sh,
                                       grad_weights, workspace, n_edges, st, n_nodes);
            if (rc != E3_OK) return rc;
            E3_CUDA_TRY(cudaEventRecord(plan->ov_ev[k], st));
            E3_CUDA_TRY(cudaStreamWaitEvent(plan->side_stream, plan->ov_ev[k], 0));
            rc = launch_dx_reduce((const float *)workspace, perm_s, col_ptr, n_nodes, plan->in_size(), grad_feats, plan->side_stream, receivers, r_lo, r_hi);
            if (rc != E3_OK) return rc;
            r_lo = r_hi;
        }
        if (plan->mid_event) E3_CUDA_TRY(cudaEventRecord(plan->mid_event, st));
        const int roles = gsh_parts(plan);
        if (roles > 0) {
            const int rc = launch_gsh_reduce(reinterpret_cast<const float *>(reinterpret_cast<const char *>(workspace) + gsh_parts_offset(plan, n_edges)),
                                             roles, n_edges * plan->sh_dim, grad_sh, st);
            if (rc != E3_OK) return rc;
        }
        E3_CUDA_TRY(cudaEventRecord(plan->ov_ev[e3_plan::kMaxOverlap], plan->side_stream));  // join
        E3_CUDA_TRY(cudaStreamWaitEvent(st, plan->ov_ev[e3_plan::kMaxOverlap], 0));
        return E3_OK;
    }
    int rc = launch_bwd_phase1(plan, feats, sh, weights, senders, row_ptr, n_nodes, grad_out, grad_sh, grad_weights, workspace, n_edges, st);
    if (rc != E3_OK) return rc;
    if (plan->mid_event) E3_CUDA_TRY(cudaEventRecord(plan->mid_event, st));
    return launch_bwd_phase2(plan, perm_s, col_ptr, n_edges, n_nodes, grad_feats, grad_sh, workspace, st);
}

// ---------------------------------------------------------------------------------------------
// NEXT-2: second-order VJP.  The forward is trilinear, so every term of the VJP-of-VJP is a first-order
// call with one operand replaced by its cotangent (oracle: orc_tp_vjp_vjp and its composition pins):
//   gg = T(vx,Y,w) + T(x,vY,w) + T(x,Y,vw)
//   (-,   dY1, dw1) = VJP(vx, Y,  w ; g)      (dx2, -,   dw2) = VJP(x, vY, w ; g)      (dx3, dY3, -) = VJP(x, Y, vw ; g)
//   gx = dx2 + dx3,  gY = dY1 + dY3,  gw = dw1 + dw2
// A NULL cotangent is zero and drops its calls; a NULL output is not computed.
// ---------------------------------------------------------------------------------------------
extern "C" size_t e3_vjp_vjp_workspace_bytes(const e3_plan *plan, int64_t n_edges, int32_t n_nodes)
{
    if (!plan || n_edges < 0 || n_nodes < 0) return 0;
    auto up = [](size_t b) { return ((b + 255) / 256) * 256; };
    return up(e3_bwd_workspace_bytes(plan, n_edges, n_nodes)) + up((size_t)n_nodes * plan->out_size() * 4) + up((size_t)n_nodes * plan->in_size() * 4) +
           up((size_t)n_edges * plan->sh_dim * 4) + up((size_t)n_edges * plan->w_size() * 4) + 256;
}

extern "C" int e3_tp_scatter_vjp_vjp(const e3_plan *plan, const void *feats, const void *sh, const void *weights, const int32_t *senders,
                                     const int32_t *receivers, const int32_t *row_ptr, const int32_t *perm_s, const int32_t *col_ptr, int64_t n_edges,
                                     int32_t n_nodes, const float *grad_out, const float *v_feats, const float *v_sh, const float *v_weights,
                                     float *gg_out, float *g_feats, float *g_sh, float *g_weights, void *workspace, size_t workspace_bytes, e3_stream stream)
{
    (void)receivers;
    if (!plan || n_edges < 0 || n_nodes < 0 || !row_ptr || !col_ptr || (n_nodes > 0 && (!feats || !grad_out)) ||
        (n_edges > 0 && (!sh || !weights || !senders || !perm_s))) {
        set_error("e3_tp_scatter_vjp_vjp: bad arguments");
        return E3_ERR_INVALID_ARG;
    }
    if (plan->dtype != E3_F32) { set_error("e3_tp_scatter_vjp_vjp: E3_F32 plans only (cotangents stand in for operands)"); return E3_ERR_UNSUPPORTED; }
    const void *ptrs[] = { feats, sh, weights, grad_out, v_feats, v_sh, v_weights, gg_out, g_feats, g_sh, g_weights, workspace };
    for (const void *q : ptrs) if (!aligned16(q)) { set_error("e3_tp_scatter_vjp_vjp: tensor pointers must be 16-byte aligned"); return E3_ERR_INVALID_ARG; }
    if (!workspace || workspace_bytes < e3_vjp_vjp_workspace_bytes(plan, n_edges, n_nodes)) {
        set_error("e3_tp_scatter_vjp_vjp: workspace too small (need %zu bytes)", e3_vjp_vjp_workspace_bytes(plan, n_edges, n_nodes));
        return E3_ERR_WORKSPACE;
    }
    if (n_nodes == 0) return E3_OK;
    cudaStream_t st = S(stream);
    auto up = [](size_t b) { return ((b + 255) / 256) * 256; };
    const size_t n_out = (size_t)n_nodes * plan->out_size(), n_in = (size_t)n_nodes * plan->in_size();
    const size_t n_sh = (size_t)n_edges * plan->sh_dim, n_w = (size_t)n_edges * plan->w_size();
    char *wp = (char *)workspace;
    void *bws = wp; wp += up(e3_bwd_workspace_bytes(plan, n_edges, n_nodes));
    float *t_out = (float *)wp; wp += up(n_out * 4);
    float *t_in = (float *)wp; wp += up(n_in * 4);
    float *t_sh = (float *)wp; wp += up(n_sh * 4);
    float *t_w = (float *)wp;
    int rc = E3_OK;
    // ---- gg: tangent of the forward
    if (gg_out) {
        bool first = true;
        const void *ops[3][3] = { { v_feats, sh, weights }, { feats, v_sh, weights }, { feats, sh, v_weights } };
        const bool have[3] = { v_feats != nullptr, v_sh != nullptr, v_weights != nullptr };
        for (int k = 0; k < 3 && rc == E3_OK; ++k) {
            if (!have[k] || (k > 0 && n_edges == 0)) continue;
            rc = launch_fwd(plan, ops[k][0], ops[k][1], ops[k][2], senders, row_ptr, n_nodes, first ? gg_out : t_out, st);
            if (rc == E3_OK && !first) rc = launch_add_inplace(gg_out, t_out, (long long)n_out, st);
            first = false;
        }
        if (first) E3_CUDA_TRY(cudaMemsetAsync(gg_out, 0, n_out * 4, st));
    }
    if (rc != E3_OK) return rc;
    // ---- first-order VJPs with one operand replaced
    bool gx_set = false, gy_set = false, gw_set = false;
    auto vjp = [&](const void *xa, const void *ya, const void *wa, float *dx_dst, float *dy_dst, float *dw_dst) -> int {
        // outputs not wanted go to the temporaries (the kernels always produce grad_feats and grad_sh; grad_weights may be NULL)
        int r2 = launch_bwd_phase1(plan, xa, ya, wa, senders, row_ptr, n_nodes, grad_out, dy_dst ? dy_dst : t_sh, dw_dst, bws, n_edges, st);
        if (r2 == E3_OK) r2 = launch_bwd_phase2(plan, perm_s, col_ptr, n_edges, n_nodes, dx_dst ? dx_dst : t_in, dy_dst ? dy_dst : t_sh, bws, st);
        return r2;
    };
    if (n_edges > 0) {
        if (v_feats && (g_sh || g_weights)) {                         // VJP(vx, Y, w): dY1 -> gY, dw1 -> gw
            rc = vjp(v_feats, sh, weights, nullptr, g_sh, g_weights);
            if (rc != E3_OK) return rc;
            gy_set = g_sh != nullptr; gw_set = g_weights != nullptr;
        }
        if (v_sh && (g_feats || g_weights)) {                         // VJP(x, vY, w): dx2 -> gx, dw2 -> gw (+)
            float *dwd = g_weights ? (gw_set ? t_w : g_weights) : nullptr;
            rc = vjp(feats, v_sh, weights, g_feats, nullptr, dwd);
            if (rc == E3_OK && g_weights && gw_set) rc = launch_add_inplace(g_weights, t_w, (long long)n_w, st);
            if (rc != E3_OK) return rc;
            gx_set = g_feats != nullptr; gw_set = gw_set || g_weights != nullptr;
        }
        if (v_weights && (g_feats || g_sh)) {                         // VJP(x, Y, vw): dx3 -> gx (+), dY3 -> gY (+)
            float *dxd = g_feats ? (gx_set ? t_in : g_feats) : nullptr;
            float *dyd = g_sh ? (gy_set ? t_sh : g_sh) : nullptr;
            rc = vjp(feats, sh, v_weights, dxd, dyd, nullptr);
            if (rc == E3_OK && g_feats && gx_set) rc = launch_add_inplace(g_feats, t_in, (long long)n_in, st);
            if (rc == E3_OK && g_sh && gy_set) rc = launch_add_inplace(g_sh, t_sh, (long long)n_sh, st);
            if (rc != E3_OK) return rc;
            gx_set = gx_set || g_feats != nullptr; gy_set = gy_set || g_sh != nullptr;
        }
    }
    if (g_feats && !gx_set) E3_CUDA_TRY(cudaMemsetAsync(g_feats, 0, n_in * 4, st));
    if (g_sh && !gy_set && n_sh) E3_CUDA_TRY(cudaMemsetAsync(g_sh, 0, n_sh * 4, st));
    if (g_weights && !gw_set && n_w) E3_CUDA_TRY(cudaMemsetAsync(g_weights, 0, n_w * 4, st));
    return E3_OK;
}

extern "C" int e3_sh_bwd_bwd(const e3_plan *plan, const float *vec, const float *grad_sh, const float *u, int64_t n_edges, float *g_vec,
                             float *g_sh, e3_stream stream)
{
    if (!plan || n_edges < 0 || (n_edges > 0 && (!vec || !u || (g_vec && !grad_sh)))) { set_error("e3_sh_bwd_bwd: bad arguments"); return E3_ERR_INVALID_ARG; }
    return launch_sh_bwd_bwd(plan->sh_lmax, vec, grad_sh, u, n_edges, g_vec, g_sh, S(stream));
}

extern "C" int e3_profile_set_mid_event(e3_plan *plan, void *cuda_event)
{
    if (!plan) { set_error("plan is NULL"); return E3_ERR_INVALID_ARG; }
    plan->mid_event = reinterpret_cast<cudaEvent_t>(cuda_event);
    return E3_OK;
}

extern "C" int e3_measure_fp32_peak(double *tflops, double ms_target, e3_stream stream)
{
    if (!tflops || !(ms_target > 0.0)) { set_error("e3_measure_fp32_peak: bad arguments"); return E3_ERR_INVALID_ARG; }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); set_error("no CUDA device"); return E3_ERR_CUDA; }
    return measure_fp32_peak(tflops, ms_target, S(stream));
}

// ---------------------------------------------------------------------------------------------
// host-buffer session
// ---------------------------------------------------------------------------------------------
struct e3_session {
    static constexpr int kMaxChunks = 64;
    const e3_plan *plan = nullptr;
    int64_t max_edges = 0;
    int32_t max_nodes = 0;
    cudaStream_t stream = nullptr, stream_in = nullptr, stream_out = nullptr;
    cudaEvent_t ev_small = nullptr, ev_done = nullptr, ev_in[kMaxChunks] = {}, ev_fwd[kMaxChunks] = {}, ev_bwd[kMaxChunks] = {};
    float *vec = nullptr, *out = nullptr, *gout = nullptr, *gfeats = nullptr, *gsh = nullptr, *gvec = nullptr, *forces = nullptr;
    void *feats = nullptr, *sh = nullptr, *weights = nullptr, *gweights = nullptr, *ws = nullptr, *gws = nullptr;
    int32_t *snd = nullptr, *rcv = nullptr, *row_ptr = nullptr, *perm_s = nullptr, *col_ptr = nullptr;
    size_t ws_bytes = 0, gws_bytes = 0;
};

extern "C" int e3_session_destroy(e3_session *s)
{
    if (!s) return E3_OK;
    void *ptrs[] = { s->vec, s->out, s->gout, s->gfeats, s->gsh, s->gvec, s->forces, s->feats, s->sh, s->weights, s->gweights,
                     s->ws, s->gws, s->snd, s->rcv, s->row_ptr, s->perm_s, s->col_ptr };
    for (void *p : ptrs) if (p) cudaFree(p);
    for (int k = 0; k < e3_session::kMaxChunks; ++k) {
        if (s->ev_in[k]) cudaEventDestroy(s->ev_in[k]);
        if (s->ev_fwd[k]) cudaEventDestroy(s->ev_fwd[k]);
        if (s->ev_bwd[k]) cudaEventDestroy(s->ev_bwd[k]);
    }
    if (s->ev_small) cudaEventDestroy(s->ev_small);
    if (s->ev_done) cudaEventDestroy(s->ev_done);
    if (s->stream) cudaStreamDestroy(s->stream);
    if (s->stream_in) cudaStreamDestroy(s->stream_in);
    if (s->stream_out) cudaStreamDestroy(s->stream_out);
    delete s;
    return E3_OK;
}

extern "C" int e3_session_create(e3_session **session, const e3_plan *plan, int64_t max_edges, int32_t max_nodes)
{
    if (!session || !plan || max_edges < 0 || max_nodes < 0) { set_error("e3_session_create: bad arguments"); return E3_ERR_INVALID_ARG; }
    *session = nullptr;
    e3_session *s = new (std::nothrow) e3_session();
    if (!s) { set_error("out of host memory"); return E3_ERR_INVALID_ARG; }
    s->plan = plan; s->max_edges = max_edges; s->max_nodes = max_nodes;
    const size_t E = (size_t)max_edges + 1, N = (size_t)max_nodes + 1, es = esize(plan);
    const size_t in_row = (size_t)plan->in_size(), out_row = (size_t)plan->out_size(), w_row = (size_t)plan->w_size();
    s->ws_bytes = e3_bwd_workspace_bytes(plan, max_edges, max_nodes);
    s->gws_bytes = graph_workspace_bytes(max_edges, max_nodes);
    cudaError_t e = cudaStreamCreateWithFlags(&s->stream, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&s->stream_in, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&s->stream_out, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&s->ev_small, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&s->ev_done, cudaEventDisableTiming);
    for (int k = 0; k < e3_session::kMaxChunks && e == cudaSuccess; ++k) {
        e = cudaEventCreateWithFlags(&s->ev_in[k], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&s->ev_fwd[k], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&s->ev_bwd[k], cudaEventDisableTiming);
    }
#define SALLOC(ptr, bytes) if (e == cudaSuccess) e = cudaMalloc((void **)&(ptr), (bytes))
    SALLOC(s->vec, E * 3 * 4); SALLOC(s->gvec, E * 3 * 4); SALLOC(s->forces, N * 3 * 4);
    SALLOC(s->feats, N * in_row * es); SALLOC(s->gfeats, N * in_row * 4);
    SALLOC(s->out, N * out_row * 4); SALLOC(s->gout, N * out_row * 4);
    SALLOC(s->sh, E * plan->sh_dim * es); SALLOC(s->gsh, E * plan->sh_dim * 4);
    SALLOC(s->weights, E * w_row * es); SALLOC(s->gweights, E * w_row * es);
    SALLOC(s->ws, s->ws_bytes); SALLOC(s->gws, s->gws_bytes);
    SALLOC(s->snd, E * 4); SALLOC(s->rcv, E * 4); SALLOC(s->row_ptr, (N + 1) * 4); SALLOC(s->perm_s, E * 4); SALLOC(s->col_ptr, (N + 1) * 4);
#undef SALLOC
    if (e != cudaSuccess) { e3_session_destroy(s); return cuda_fail(e, "session allocation"); }
    *session = s;
    return E3_OK;
}

// The run is pipelined over contiguous receiver ranges ("chunks"): the weights of chunk k+1 travel host->device on one
// copy stream while chunk k is computed, and chunk k-1's `out` rows and grad_weights travel device->host on another
// (PCIe is full duplex; the weights and their gradients are > 95 % of the bytes).  Results do not depend on the chunking:
// a chunk is the same kernels, in the launch shape chosen for the whole graph, on a receiver range, and the per-sender
// reduction runs once at the end.
static int session_run_host_impl(e3_session *s, const float *vec_h, const void *feats_h, const void *weights_h,
                                   const int32_t *senders_h, const int32_t *receivers_h, int64_t n_edges, int32_t n_nodes,
                                   const float *grad_out_h, float *out_h, float *grad_feats_h, void *grad_weights_h,
                                   float *grad_vec_h, float *forces_h, int64_t *bytes_h2d, int64_t *bytes_d2h)
{
    if (!s || n_edges < 0 || n_nodes < 0 || n_edges > s->max_edges || n_nodes > s->max_nodes ||
        (n_nodes > 0 && !feats_h) || (n_edges > 0 && (!vec_h || !weights_h || !senders_h || !receivers_h))) {
        set_error("e3_session_run_host: bad arguments or sizes above the session capacity");
        return E3_ERR_INVALID_ARG;
    }
    // the index arrays are on the host: range and sortedness are checked here, before anything is launched
    // (the kernels index row_ptr / col_ptr / feats with them and the chunking below bisects receivers_h)
    for (int64_t e = 0; e < n_edges; ++e) {
        const int32_t sv = senders_h[e], rv = receivers_h[e];
        if (sv < 0 || sv >= n_nodes || rv < 0 || rv >= n_nodes) {
            set_error("e3_session_run_host: edge %lld has an index out of range [0, %d)", (long long)e, (int)n_nodes);
            return E3_ERR_INVALID_ARG;
        }
        if (e > 0 && rv < receivers_h[e - 1]) {
            set_error("e3_session_run_host: receivers are not sorted ascending (edge %lld)", (long long)e);
            return E3_ERR_UNSORTED;
        }
    }
    const e3_plan *pl = s->plan;
    const size_t E = (size_t)n_edges, N = (size_t)n_nodes, es = esize(pl);
    const size_t in_row = (size_t)pl->in_size(), out_row = (size_t)pl->out_size(), w_row = (size_t)pl->w_size();
    cudaStream_t st = s->stream, sin = s->stream_in, sout = s->stream_out;
    int64_t up = 0, down = 0;
#define H2D(stream_, dst, src, bytes) do { if ((bytes) > 0) { E3_CUDA_TRY(cudaMemcpyAsync((dst), (src), (bytes), cudaMemcpyHostToDevice, (stream_))); up += (int64_t)(bytes); } } while (0)
#define D2H(stream_, dst, src, bytes) do { if ((dst) && (bytes) > 0) { E3_CUDA_TRY(cudaMemcpyAsync((dst), (src), (bytes), cudaMemcpyDeviceToHost, (stream_))); down += (int64_t)(bytes); } } while (0)
    // small inputs first
    H2D(sin, s->snd, senders_h, E * 4); H2D(sin, s->rcv, receivers_h, E * 4); H2D(sin, s->vec, vec_h, E * 12);
    H2D(sin, s->feats, feats_h, N * in_row * es);
    if (grad_out_h) H2D(sin, s->gout, grad_out_h, N * out_row * 4);
    E3_CUDA_TRY(cudaEventRecord(s->ev_small, sin));
    E3_CUDA_TRY(cudaStreamWaitEvent(st, s->ev_small, 0));
    int rc = launch_graph_prepare(s->snd, s->rcv, n_edges, n_nodes, s->row_ptr, s->perm_s, s->col_ptr, s->gws, s->gws_bytes, 0, st);
    if (rc == E3_OK) rc = e3_sh_fwd(pl, s->vec, n_edges, s->sh, st);
    if (rc != E3_OK) return rc;
    // receiver ranges of roughly equal edge counts (~48 MB of weights each); rows must stay 16-byte aligned under the offsets
    int n_chunks = (int)((E * w_row * es + (48u << 20) - 1) / (48u << 20));
    n_chunks = n_chunks < 1 ? 1 : (n_chunks > e3_session::kMaxChunks ? e3_session::kMaxChunks : n_chunks);
    if ((out_row * 4) % 16 != 0 || (w_row * es) % 16 != 0 || n_nodes == 0) n_chunks = 1;
    int32_t r_lo = 0;
    int n_used = 0;
    for (int k = 0; k < n_chunks && r_lo < n_nodes; ++k) {
        int32_t r_hi = n_nodes;
        if (k + 1 < n_chunks && n_edges > 0) {
            const int64_t e_target = (int64_t)((double)(k + 1) / n_chunks * (double)n_edges);
            r_hi = e_target < n_edges ? receivers_h[e_target] : n_nodes;      // receivers_h is sorted: edges of r < r_hi come first
            if (r_hi <= r_lo) continue;
        }
        // edges of receivers [r_lo, r_hi): [e_lo, e_hi) by binary search in the sorted host array
        auto lower = [&](int32_t r) { int64_t a = 0, b = n_edges; while (a < b) { int64_t m = (a + b) / 2; if (receivers_h[m] < r) a = m + 1; else b = m; } return a; };
        const int64_t e_lo = lower(r_lo), e_hi = lower(r_hi);
        const int32_t nr = r_hi - r_lo;
        H2D(sin, (char *)s->weights + (size_t)e_lo * w_row * es, (const char *)weights_h + (size_t)e_lo * w_row * es, (size_t)(e_hi - e_lo) * w_row * es);
        E3_CUDA_TRY(cudaEventRecord(s->ev_in[n_used], sin));
        E3_CUDA_TRY(cudaStreamWaitEvent(st, s->ev_in[n_used], 0));
        rc = launch_fwd(pl, s->feats, s->sh, s->weights, s->snd, s->row_ptr + r_lo, nr, s->out + (size_t)r_lo * out_row, st, n_nodes);
        if (rc != E3_OK) return rc;
        E3_CUDA_TRY(cudaEventRecord(s->ev_fwd[n_used], st));
        E3_CUDA_TRY(cudaStreamWaitEvent(sout, s->ev_fwd[n_used], 0));
        D2H(sout, out_h ? out_h + (size_t)r_lo * out_row : nullptr, s->out + (size_t)r_lo * out_row, (size_t)nr * out_row * 4);
        if (grad_out_h) {
            rc = launch_bwd_phase1(pl, s->feats, s->sh, s->weights, s->snd, s->row_ptr + r_lo, nr, s->gout + (size_t)r_lo * out_row, s->gsh,
                                   grad_weights_h ? s->gweights : nullptr, s->ws, n_edges, st, n_nodes);
            if (rc != E3_OK) return rc;
            E3_CUDA_TRY(cudaEventRecord(s->ev_bwd[n_used], st));
            E3_CUDA_TRY(cudaStreamWaitEvent(sout, s->ev_bwd[n_used], 0));
            D2H(sout, grad_weights_h ? (char *)grad_weights_h + (size_t)e_lo * w_row * es : nullptr, (char *)s->gweights + (size_t)e_lo * w_row * es,
                (size_t)(e_hi - e_lo) * w_row * es);
        }
        r_lo = r_hi;
        ++n_used;
    }
    if (grad_out_h) {
        rc = launch_bwd_phase2(pl, s->perm_s, s->col_ptr, n_edges, n_nodes, s->gfeats, s->gsh, s->ws, st);
        if (rc == E3_OK) rc = e3_sh_bwd(pl, s->vec, s->gsh, n_edges, s->gvec, st);
        if (rc == E3_OK && forces_h) rc = e3_force_reduce(s->gvec, s->row_ptr, s->perm_s, s->col_ptr, n_edges, n_nodes, s->forces, st);
        if (rc != E3_OK) return rc;
        E3_CUDA_TRY(cudaEventRecord(s->ev_done, st));
        E3_CUDA_TRY(cudaStreamWaitEvent(sout, s->ev_done, 0));
        D2H(sout, grad_feats_h, s->gfeats, N * in_row * 4);
        D2H(sout, grad_vec_h, s->gvec, E * 12);
        D2H(sout, forces_h, s->forces, N * 12);
    }
#undef H2D
#undef D2H
    E3_CUDA_TRY(cudaStreamSynchronize(sin));
    E3_CUDA_TRY(cudaStreamSynchronize(st));
    E3_CUDA_TRY(cudaStreamSynchronize(sout));
    if (bytes_h2d) *bytes_h2d = up;
    if (bytes_d2h) *bytes_d2h = down;
    return E3_OK;
}

extern "C" int e3_session_run_host(e3_session *s, const float *vec_h, const void *feats_h, const void *weights_h,
                                   const int32_t *senders_h, const int32_t *receivers_h, int64_t n_edges, int32_t n_nodes,
                                   const float *grad_out_h, float *out_h, float *grad_feats_h, void *grad_weights_h,
                                   float *grad_vec_h, float *forces_h, int64_t *bytes_h2d, int64_t *bytes_d2h)
{
    const int rc = session_run_host_impl(s, vec_h, feats_h, weights_h, senders_h, receivers_h, n_edges, n_nodes, grad_out_h, out_h,
                                         grad_feats_h, grad_weights_h, grad_vec_h, forces_h, bytes_h2d, bytes_d2h);
    if (rc != E3_OK && s) {      // no asynchronous copy may still touch the caller's host buffers after a failing return
        cudaStreamSynchronize(s->stream_in);
        cudaStreamSynchronize(s->stream);
        cudaStreamSynchronize(s->stream_out);
        cudaGetLastError();
    }
    return rc;
}
