// Internal declarations shared by the translation units of libe3b200.so (never installed).
#pragma once
#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/e3b200.h"

namespace e3 {

constexpr int kMaxL = 3;      // highest degree supported anywhere (irreps, SH)
constexpr int kMaxShDim = 16;

// thread-local error detail -------------------------------------------------------------------
void set_error(const char *fmt, ...);
const char *get_error();
int cuda_fail(cudaError_t e, const char *what);     // records text, returns E3_ERR_CUDA

#define E3_CUDA_TRY(expr)                                          \
    do {                                                           \
        cudaError_t e3_err__ = (expr);                             \
        if (e3_err__ != cudaSuccess) return ::e3::cuda_fail(e3_err__, #expr); \
    } while (0)

// one non-zero of a real Clebsch-Gordan tensor (indices 0-based: m_true + l)
struct Nz { int m1, m2, m3; double c; };

struct PathInfo {
    int i_in, l_sh, i_out;     // as given by the caller
    int l1, l2, l3;
    int in_off, out_off;       // first row (in units of C-wide rows) of the irrep block in a node row
    std::vector<Nz> nz;        // sparse real CG, ordered m1, m2, m3
    int nzM;                   // structurally non-zero (m1, m3) pairs
};

// A forward "role": a set of output irreps (and every path feeding them) owned by one warp.
struct Role {
    std::vector<int> out_irreps;
    std::vector<int> paths;
    int rows;                  // accumulator rows (sum of 2l3+1 over out_irreps)
    double cost;
};

struct JitKernel {
    std::string name;
    std::string source;
    std::vector<char> cubin;
    int regs = 0, spill = 0, smem = 0, threads = 0;
    int smem_dyn = 0;          // dynamic shared memory per CTA (operand rings)
    cudaLibrary_t lib = nullptr;
    cudaKernel_t fn = nullptr;
};

}  // namespace e3

struct e3_plan {
    std::vector<e3_irrep> irreps_in, irreps_out;
    std::vector<e3::PathInfo> paths;
    int sh_lmax = 0, sh_dim = 0, in_dim = 0, out_dim = 0, C = 0;
    e3_dtype dtype = E3_F32;
    int nnz_total = 0;
    // launch geometry chosen by the code generator
    int K = 1;                 // channels per lane
    int nchb = 1;              // channel blocks of 32*K
    std::vector<e3::Role> roles;
    int fwd_warps = 4, bwd_warps = 4;
    int ring = 0;              // 1: cp.async operand rings, 0: plain loads (odd shapes)
    int v2 = 0;                // 1: second-generation kernels (factored form, 4 channels per lane, codegen2.cpp)
    int lpe = 32, eps = 1;     // v2: lanes per edge (C/4, at most 32) and edges per warp step (32/lpe)
    int nchb2 = 1;             // v2: channel blocks of 128
    int fwd_depth = 4;         // forward ring stages (power of two); the backward ring has one rolling stage
    int fwd_depth_max = 6;     // v2 forward: roles with small stages deepen their ring up to this many stages
    int fwd_chunk = 16;        // CTAs per (chunk, role): CTA order is chunk-major, then role
    int fwd_minb = 4, bwd_minb = 2;        // __launch_bounds__ min blocks per SM
    int bwd_v2 = 0;            // 1: second-generation backward (codegen2.cpp)
    int bwd_r = 0;             // v2 backward: weights ring holds 1/bwd_r of a unit (0 = choose; set by the generator)
    int bwd_nroles = 1;        // v2 backward: roles (runs of input irreps) per receiver; grad_sh is summed over roles afterwards
    int bwd_role_cost = 0;     // v2 backward: cost target of one role in packed operations (0 = default)
    int bwd_chunk = 4096;      // v2 backward: receivers per chunk (CTA order is chunk-major, then role)
    int bwd_depth = 0;         // v2 backward: ring stages per warp (units in flight); 0 = choose
    int bwd_split = 0;         // v2 backward: CTAs per receiver (0 = choose at launch from the grid size)
    int fwd_split = 0;         // v2 forward: warps sharing one (receiver, role) (0 = choose at launch)
    // third-generation forward (codegen2.cpp gen_forward_v3): a CTA = the roles ("team") of ONE receiver; operands arrive by
    // TMA bulk copies (cp.async.bulk + mbarrier), the team's sender rows once per edge instead of once per role
    int fwd_v3 = 0;
    int fwd_tw = 3;            // warps (roles) per team at most
    int fwd_v3_depth = 0;      // ring stages per team (0 = choose)
    int fwd_v3_bulk = 0;       // 1: operands by cp.async.bulk (one elected lane per warp; measured 4.5x slower on config 4: the copies are
                               // 256 B - 1.8 KB each); 0: per-lane 16-byte cp.async completing on the stage's mbarrier
    int fwd_v3_lag = 1;        // a stage is refilled `lag` steps after it was consumed (slack between the team's warps)
    int fwd_v3_stage = 0, fwd_v3_part = 0, fwd_v3_bar = 1024;   // bytes: one ring stage, one sub-team's partial sums, the barrier block
    int fwd_v3_chunk = 1 << 30;   // receivers per (chunk, team): CTA order is chunk-major, then team (default: team-major, one team's code per SM)
    std::vector<std::vector<int>> teams;     // role indices per team
    void *zeros = nullptr;     // device buffer of zeros (source of the operands of a step's missing edges)
    size_t zeros_bytes = 0;
    int wait_all = 0;          // checking aid (E3_TUNE wait_all=1): every cp.async wait drains all outstanding groups, so a result that differs
                               // from the normal build would expose a static wait count that is too loose (tests/test_gpu_gaps.py)
    int fwd_ctas_per_sm = 2, bwd_ctas_per_sm = 2;   // measured residency (occupancy API) of the loaded kernels
    int n_sm = 148;            // SM count of the device the plan was created on
    e3::JitKernel fwd, bwd;
    cudaEvent_t mid_event = nullptr;   // profiling aid, see e3_profile_set_mid_event
    // VJP overlap: the first phase is launched in `bwd_overlap` receiver chunks and the per-sender reduction of the
    // senders a chunk completes runs on a side stream while the next chunk computes.  -1 / 0 = off (the default: measured slower), K = K chunks.
    int bwd_overlap = -1;
    static constexpr int kMaxOverlap = 16;
    cudaStream_t side_stream = nullptr;
    cudaEvent_t ov_ev[kMaxOverlap + 1] = {};

    // Element layout of a node row / a weights row.  A regular plan (all multiplicities equal to C) has its irrep blocks back to
    // back, (2l+1)*C elements each.  NEXT-4, unequal multiplicities: the plan is a COMPOSITE of one sub-plan per multiplicity
    // class (`subs`, each a regular generated plan over the irreps and paths of that class) whose kernels address the rows of the
    // whole plan: strides and block offsets are overridden by the vectors below (empty = regular layout).
    std::vector<e3_plan *> subs;                 // composite: one sub-plan per multiplicity class (owned)
    std::vector<std::pair<int, int>> path_map;   // composite: path p of the caller = path .second of subs[.first]
    int in_size_all = 0, out_size_all = 0, w_size_all = 0;   // composite: elements per row of the whole plan
    int in_stride = 0, out_stride = 0, w_stride = 0;         // sub-plan: row strides in elements (0 = regular)
    std::vector<int> in_base, out_base, w_base;              // sub-plan: element offset of input irrep i / output irrep i / path p
    std::vector<std::pair<int, int>> zero_in;                // sub-plan: (offset, length) element runs of the whole input row that no path of
                                                             // any class reads; its backward writes their zero rows of the per-edge workspace
    int in_size() const { return !subs.empty() ? in_size_all : (in_stride ? in_stride : in_dim * C); }
    int out_size() const { return !subs.empty() ? out_size_all : (out_stride ? out_stride : out_dim * C); }
    int w_size() const { return !subs.empty() ? w_size_all : (w_stride ? w_stride : (int)paths.size() * C); }
    int xoff(int i_in, int m1) const
    {
        if (!in_base.empty()) return in_base[i_in] + m1 * C;
        int off = 0;
        for (int i = 0; i < i_in; ++i) off += 2 * irreps_in[i].l + 1;
        return (off + m1) * C;
    }
    int ooff(int i_out, int m3) const
    {
        if (!out_base.empty()) return out_base[i_out] + m3 * C;
        int off = 0;
        for (int i = 0; i < i_out; ++i) off += 2 * irreps_out[i].l + 1;
        return (off + m3) * C;
    }
    int woff(int p) const { return w_base.empty() ? p * C : w_base[p]; }
};

namespace e3 {

// plan.cu
double cg_real_host(int l1, int l2, int l3, int m1, int m2, int m3);   // same routine as the device planner kernel
int plan_build_tables(e3_plan &pl, const e3_irrep *irreps_in, int n_in, int sh_lmax, const e3_irrep *irreps_out,
                      int n_out, const e3_path *paths, int n_paths, e3_dtype dtype, bool cg_on_device);
void plan_make_roles(e3_plan &pl);
bool plan_is_composite(const e3_irrep *irreps_in, int n_in, const e3_irrep *irreps_out, int n_out);   // multiplicities differ
int plan_build_composite(e3_plan &pl, const e3_irrep *irreps_in, int n_in, int sh_lmax, const e3_irrep *irreps_out, int n_out,
                         const e3_path *paths, int n_paths, e3_dtype dtype, bool cg_on_device);

// codegen.cpp
std::string gen_forward_source(e3_plan &pl);    // also sets pl.fwd.smem_dyn
std::string gen_backward_source(e3_plan &pl);   // also sets pl.bwd.smem_dyn

// codegen2.cpp (second generation; used when v2_eligible)
bool v2_eligible(const e3_plan &pl);
std::string gen_forward_v2(e3_plan &pl);
std::string gen_backward_v2(e3_plan &pl);  // also sets pl.bwd.smem_dyn, pl.bwd_r
bool v3_eligible(const e3_plan &pl);
std::string gen_forward_v3(e3_plan &pl);   // sets pl.fwd.smem_dyn (for fsplit = 1), pl.fwd_v3_depth

// jit.cpp
int jit_compile(JitKernel &k, const std::string &file_hint);   // NVRTC -> cubin (+regs/spill from the ptxas log)
int jit_load(JitKernel &k);                                    // cubin -> cudaKernel_t (needs a device)
void jit_unload(JitKernel &k);

// kernels.cu (statically compiled kernels)
int launch_sh_fwd(int lmax, e3_dtype dt, const float *vec, int64_t E, void *sh, cudaStream_t st);
int launch_sh_bwd(int lmax, const float *vec, const float *gsh, int64_t E, float *gvec, cudaStream_t st);
size_t graph_workspace_bytes(int64_t E, int32_t N);
int launch_graph_prepare(const int32_t *snd, const int32_t *rcv, int64_t E, int32_t N, int32_t *row_ptr,
                         int32_t *perm_s, int32_t *col_ptr, void *ws, size_t ws_bytes, int validate, cudaStream_t st);
int launch_force_reduce(const float *gvec, const int32_t *row_ptr, const int32_t *perm_s, const int32_t *col_ptr,
                        int64_t E, int32_t N, float *forces, cudaStream_t st);
int launch_dx_reduce(const float *dxe, const int32_t *perm_s, const int32_t *col_ptr, int32_t N, int row_len,
                     float *dx, cudaStream_t st, const int32_t *receivers = nullptr, int32_t r_lo = 0, int32_t r_hi = 0);
int launch_gsh_reduce(const float *parts, int n_parts, int64_t n, float *gsh, cudaStream_t st);
int measure_fp32_peak(double *tflops, double ms_target, cudaStream_t st);
int launch_sh_bwd_bwd(int lmax, const float *vec, const float *gsh, const float *u, int64_t E, float *g_vec, float *g_sh, cudaStream_t st);
int launch_add_inplace(float *dst, const float *src, long long n, cudaStream_t st);
int launch_scan_i32(int32_t *ptr, int32_t n, int32_t *cursor, cudaStream_t st);   // ptr[0..n) -> inclusive scan in place; cursor[i] = ptr[i], i < n-1
int launch_cg_planner(const int *triples /*[n,3] host*/, int n, std::vector<std::vector<double>> &dense_out);

}  // namespace e3
