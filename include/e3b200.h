/*
 * e3b200.h -- C ABI of the B200-native fused Clebsch-Gordan tensor product + scatter library
 * (the data-parallel hot path of the e3j backend of arxiv 2605.22698, "mlip v2").
 *
 * The paper only NAMES the operation: PAPER.md L72-L74 (section 4: MACE and NequIP "rely on the
 * Clebsch-Gordan Tensor Product ... a significant computational bottleneck"), L82 ("fusion of
 * the message passing kernel" is the authors' open item), L66 (the Graph class computes edge
 * vectors from positions and connectivity), L44 (CG formalism).  It prints no formula, so every
 * convention below is a reading fixed in SURVEY.md section 8(c) / DESIGN.md (A1..A18); each
 * entry point cites the reading that defines what it computes.
 *
 * General rules
 *  - Plain C types only.  Every pointer is a DEVICE pointer owned by the caller unless its
 *    name ends in _h / it is documented as host.  The library never frees or keeps caller
 *    memory, never allocates on the hot path, and launches only on the given stream.
 *  - `e3_stream` is a cudaStream_t passed as an opaque pointer (NULL = legacy default stream).
 *  - No call synchronises the stream except where stated (e3_graph_prepare with validate != 0,
 *    e3_plan_create, the e3_session_* host-buffer calls).
 *  - Every function returns an int status (E3_OK == 0).  e3_last_error() returns a
 *    thread-local detail string (NVRTC log, CUDA error text) for the last failing call.
 *  - Layouts (reading A7): a node row is the concatenation of its irrep blocks in irreps order;
 *    inside a block the element index is m*C + u, m = 0..2l (i.e. m_true + l), u = channel
 *    (channel fastest).  SH rows are indexed l*l + l + m_true.  Weights are [(e*P + p)*C + u]
 *    (64-bit offsets).  All irreps of a plan share one multiplicity C ("uvu", reading A8).
 *  - dtype (reading A12): E3_F32 stores feats, sh, weights and grad_weights as float;
 *    E3_BF16 stores those four as bfloat16 (round-to-nearest-even) and everything else
 *    (out, grad_out, grad_feats, grad_sh, vec, grad_vec, forces, accumulators) as float.
 *  - There is no CPU fallback anywhere: without a CUDA device every compute call returns
 *    E3_ERR_CUDA.
 */
#ifndef E3B200_H
#define E3B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct e3_plan e3_plan;          /* opaque, immutable after creation, thread-safe for launches */
typedef struct e3_session e3_session;    /* opaque, owns device buffers for the host-buffer entry point */
typedef void *e3_stream;                 /* cudaStream_t */

typedef struct { int l; int parity; /* +1 even, -1 odd */ int mul; } e3_irrep;
typedef struct { int i_in; int l_sh; int i_out; } e3_path;   /* indices into irreps_in / irreps_out */
typedef enum { E3_F32 = 0, E3_BF16 = 1 } e3_dtype;

enum {
    E3_OK = 0,
    E3_ERR_INVALID_ARG = 1,   /* null pointer, negative size, index out of range                     */
    E3_ERR_BAD_PATH = 2,      /* triangle rule, parity rule or irrep index violated                  */
    E3_ERR_UNSUPPORTED = 3,   /* l > 3, unequal multiplicities not multiples of 4, odd row alignment */
    E3_ERR_UNSORTED = 4,      /* receivers not ascending (only when validation was requested)        */
    E3_ERR_CUDA = 5,          /* CUDA runtime error or no device                                     */
    E3_ERR_JIT = 6,           /* run-time specialisation (NVRTC) of the plan's kernels failed        */
    E3_ERR_WORKSPACE = 7      /* workspace pointer NULL or too small                                 */
};

const char *e3_status_string(int status);
const char *e3_last_error(void);

/* ---------------------------------------------------------------------------------------------
 * Path table helper (host only).  Reading A5/A6: every (i_in, l2 <= sh_lmax, l3) with
 * |l1-l2| <= l3 <= min(l1+l2, out_lmax), output parity p1*(-1)^l2 (pseudotensor outputs included
 * unless natural_parity_only), ordered by i_in, then l2, then l3; each path gets its own output
 * irrep (multiplicity of its input).  Call with out == NULL / paths == NULL to query the counts.
 * -------------------------------------------------------------------------------------------*/
int e3_all_paths(const e3_irrep *irreps_in, int n_in, int sh_lmax, int out_lmax, int natural_parity_only,
                 e3_irrep *irreps_out, int *n_out, e3_path *paths, int *n_paths);

/* ---------------------------------------------------------------------------------------------
 * Plan.  Validates the path table (E3_ERR_BAD_PATH), computes the real
 * Clebsch-Gordan tensors of all paths ON THE DEVICE in fp64 (Racah closed form + real-basis
 * change, reading A4), compacts them to sparse (m1,m2,m3,coef) lists and specialises the
 * forward and VJP kernels for this plan (coefficients become FFMA immediates).  Needs a device;
 * synchronises; takes O(seconds) once.  A path whose i_out is shared with another path ADDS
 * into that block (A6).  Limits: l <= 3 everywhere.
 * Multiplicities (NEXT-4, NequIP's `64x0e + 64x0o + 32x1o + 32x1e + 32x2e + 32x2o`): when all
 * irreps have the same multiplicity C the layouts are those of A7/A8.  Otherwise every multiplicity must be a multiple of 4, a
 * path's input and output irrep must have the same multiplicity (a channelwise path keeps it; E3_ERR_BAD_PATH otherwise), and
 * the layouts are: node row = irrep blocks back to back, block i = (2l_i+1) x mul_i values at index m*mul_i + u; weights row =
 * mul(path) values per path, paths back to back (e3_plan_sizes returns the three row lengths).  Such a plan runs one generated
 * kernel pair per multiplicity class over the same rows; every entry point below accepts it.
 * Environment: E3_TUNE="key=value,..." overrides launch-shape heuristics (never results);
 * E3_JIT_CACHE=0 disables the compiled-kernel cache (speed only).  The cache lives in a per-user directory of mode 0700
 * ($E3_JIT_DIR, else $XDG_CACHE_HOME/e3b200_jit, else /tmp/e3b200_jit_<uid>; refused if not owned by the caller or
 * group/world-writable); a hit must match two 64-bit hashes of (compile options + source), the stored source byte for
 * byte, and the cubin's recorded length and checksum.
 * -------------------------------------------------------------------------------------------*/
int e3_plan_create(e3_plan **plan, const e3_irrep *irreps_in, int n_in, int sh_lmax,
                   const e3_irrep *irreps_out, int n_out, const e3_path *paths, int n_paths, e3_dtype dtype);
int e3_plan_destroy(e3_plan *plan);
/* in_dim = sum(2l+1) over irreps_in, sh_dim = (sh_lmax+1)^2, out_dim likewise over irreps_out,
 * weights_per_edge = n_paths * C, nnz_total = number of non-zero real CG coefficients. */
int e3_plan_dims(const e3_plan *plan, int *in_dim, int *sh_dim, int *out_dim, int *weights_per_edge, int *nnz_total);
/* Row lengths in ELEMENTS: feats / grad_feats rows (sum (2l+1)*mul over irreps_in), out / grad_out rows (likewise over irreps_out)
 * and weights / grad_weights rows (sum of mul over paths).  Any pointer may be NULL. */
int e3_plan_sizes(const e3_plan *plan, int64_t *feats_per_node, int64_t *out_per_node, int64_t *weights_per_edge);
/* Host copy of path `path`'s sparse CG list (m indices are 0-based: m_true + l).  Pass m1 == NULL
 * to query *nnz only.  Order: m1, then m2, then m3 ascending. */
int e3_plan_get_cg(const e3_plan *plan, int path, int *m1, int *m2, int *m3, double *coef, int *nnz);
/* Launch facts of the specialised kernels: which = 0 forward, 1 backward.  Any pointer may be NULL. */
int e3_plan_kernel_info(const e3_plan *plan, int which, int *regs, int *spill_bytes, int *smem_bytes,
                        int *threads_per_block, int *n_roles, int *channels_per_lane);
/* Algorithmic work per edge of this plan, SURVEY 8(d) formulas (factored form), for roofline reports. */
int e3_plan_work(const e3_plan *plan, double *fwd_flop_per_edge, double *bwd_flop_per_edge);

/* Build-time check (host only, no device needed): generates and compiles the specialised
 * kernels exactly as e3_plan_create would, using a host evaluation of the same CG routine, and
 * reports registers / spills.  If src_path != NULL the generated CUDA source is written there
 * and the cubin beside it (src_path + ".cubin").  It computes nothing of the hot path. */
int e3_jit_check(const e3_irrep *irreps_in, int n_in, int sh_lmax, const e3_irrep *irreps_out, int n_out,
                 const e3_path *paths, int n_paths, e3_dtype dtype, const char *src_path,
                 int *fwd_regs, int *fwd_spill, int *bwd_regs, int *bwd_spill);

/* ---------------------------------------------------------------------------------------------
 * Graph preparation (readings A11/A14/A15).  Integer only, deterministic.
 * Input: receivers ascending.  Output: row_ptr[N+1] (CSR over receivers), perm_s[E] (edge ids in
 * ascending sender order, ties in ascending edge id = numpy stable argsort), col_ptr[N+1].
 * workspace: >= e3_graph_workspace_bytes(E, N) bytes of device memory.
 * validate != 0: additionally checks index ranges and sortedness; this SYNCHRONISES the stream
 * and returns E3_ERR_INVALID_ARG / E3_ERR_UNSORTED.
 * -------------------------------------------------------------------------------------------*/
size_t e3_graph_workspace_bytes(int64_t n_edges, int32_t n_nodes);
int e3_graph_prepare(const int32_t *senders, const int32_t *receivers, int64_t n_edges, int32_t n_nodes,
                     int32_t *row_ptr, int32_t *perm_s, int32_t *col_ptr,
                     void *workspace, size_t workspace_bytes, int validate, e3_stream stream);

/* ---------------------------------------------------------------------------------------------
 * Spherical harmonics (readings A1-A3).  sh[e, l*l+l+m] = Y_lm(vec_e/|vec_e|),
 * real basis, z polar, m<0 sine / m>0 cosine type, no Condon-Shortley sign, component
 * normalisation (sum_m Y_lm^2 = 2l+1): Y_1 = sqrt3 (y,z,x).  |vec| == 0 -> Y_00 = 1, rest 0,
 * gradient 0.  sh has the plan's storage dtype; grad_sh and grad_vec are float.
 *   grad_vec[e,:] = sum_lm grad_sh[e,lm] * d Y_lm(vec/|vec|) / d vec .
 * -------------------------------------------------------------------------------------------*/
int e3_sh_fwd(const e3_plan *plan, const float *vec /*[E,3]*/, int64_t n_edges, void *sh /*[E,sh_dim]*/,
              e3_stream stream);
int e3_sh_bwd(const e3_plan *plan, const float *vec, const float *grad_sh /*[E,sh_dim]*/, int64_t n_edges,
              float *grad_vec /*[E,3]*/, e3_stream stream);

/* ---------------------------------------------------------------------------------------------
 * Fused gather - tensor product - scatter, forward (readings A4-A8, A10):
 *   out[r, blk(p), m3, u] = sum_{e : receivers[e] = r} weights[e,p,u] *
 *        sum_{m1,m2} C^p[m1,m2,m3] * feats[senders[e], blk(l1(p)), m1, u] * sh[e, l2(p), m2]
 * Edges must be sorted by receiver; row_ptr from e3_graph_prepare.  Every row of out[N, out_dim*C]
 * is written (zeros for receivers without edges).  Deterministic: each (receiver, output row,
 * channel) is accumulated by one thread in ascending edge order; no atomics.
 * `receivers` is accepted for symmetry with the problem statement and may be NULL.
 * -------------------------------------------------------------------------------------------*/
int e3_tp_scatter_fwd(const e3_plan *plan, const void *feats /*[N,in_dim*C]*/, const void *sh /*[E,sh_dim]*/,
                      const void *weights /*[E,P*C]*/, const int32_t *senders, const int32_t *receivers,
                      const int32_t *row_ptr, int64_t n_edges, int32_t n_nodes, float *out, e3_stream stream);

/* ---------------------------------------------------------------------------------------------
 * VJP of the forward.  Given grad_out = dL/d out [N, out_dim*C] (float):
 *   grad_feats[s,l1,m1,u] = sum_{e : senders[e] = s} sum_p w[e,p,u] sum_{m2,m3} C^p sh[e,l2,m2] grad_out[r,p,m3,u]
 *   grad_sh[e,l2,m2]      = sum_p sum_u w[e,p,u] sum_{m1,m3} C^p feats[s,l1,m1,u] grad_out[r,p,m3,u]
 *   grad_weights[e,p,u]   = sum_{m1,m2,m3} C^p feats[s,l1,m1,u] sh[e,l2,m2] grad_out[r,p,m3,u]
 * grad_feats [N,in_dim*C] and grad_sh [E,sh_dim] are float; grad_weights has the plan's storage
 * dtype and may be NULL (skipped).  workspace: >= e3_bwd_workspace_bytes(plan, E, N) bytes; it
 * holds the per-edge grad_feats contributions that the second phase sums per sender in
 * ascending edge order (deterministic, no atomics).
 * Opt-in (E3_TUNE bwd_overlap=K at plan creation, `receivers` given): the first phase is launched in K receiver chunks on `stream` and
 * the sums of the senders each chunk completes run meanwhile on a stream owned by the plan; that stream waits for everything enqueued on
 * `stream` before the call and `stream` waits for it before the call returns, so the call behaves like a single-stream one (it can be
 * captured in a CUDA graph) and its results are bit-identical to the default path.  Measured slower on power-capped boards,
 * hence off by default.  `receivers` may be NULL.  One VJP call of a plan at a time when the overlap is on.
 * -------------------------------------------------------------------------------------------*/
size_t e3_bwd_workspace_bytes(const e3_plan *plan, int64_t n_edges, int32_t n_nodes);
int e3_tp_scatter_bwd(const e3_plan *plan, const void *feats, const void *sh, const void *weights,
                      const int32_t *senders, const int32_t *receivers, const int32_t *row_ptr,
                      const int32_t *perm_s, const int32_t *col_ptr, int64_t n_edges, int32_t n_nodes,
                      const float *grad_out, float *grad_feats, float *grad_sh, void *grad_weights,
                      void *workspace, size_t workspace_bytes, e3_stream stream);

/* Profiling aid (used by bench.py only): if `cuda_event` (a cudaEvent_t, or NULL to clear) is set,
 * e3_tp_scatter_bwd records it on its stream between its two kernels, so that the dominant first
 * phase and the per-sender reduction can be timed separately with CUDA events.  Not thread-safe. */
int e3_profile_set_mid_event(e3_plan *plan, void *cuda_event);

/* Measurement aid (used by bench.py only; SURVEY section 7 "FP32 peak is not in MEASURED_PEAKS.json"): runs a
 * register-only packed-FMA kernel (8 independent FFMA2 chains per thread, one full wave of 1024-thread CTAs) for about
 * `ms_target` milliseconds on `stream`, synchronises, and returns the achieved FP32 rate in TFLOP/s (2 flop per FMA lane)
 * in *tflops.  It is the sustained FFMA ceiling of THIS board at the clock its power cap allows, reported beside the nominal
 * 148 x 128 x 2 x 1.965 GHz peak that the roofline fractions use.  Returns E3_ERR_CUDA without a device. */
int e3_measure_fp32_peak(double *tflops, double ms_target, e3_stream stream);

/* ---------------------------------------------------------------------------------------------
 * Edge -> atom force reduction (reading A10: vec_e = pos[rcv] - pos[snd] + shift):
 *   forces[i,:] = -( sum_{e : receivers[e]=i} grad_vec[e,:] - sum_{e : senders[e]=i} grad_vec[e,:] )
 * Fixed summation order (one warp per atom, no atomics).
 * -------------------------------------------------------------------------------------------*/
int e3_force_reduce(const float *grad_vec /*[E,3]*/, const int32_t *row_ptr, const int32_t *perm_s,
                    const int32_t *col_ptr, int64_t n_edges, int32_t n_nodes, float *forces /*[N,3]*/,
                    e3_stream stream);

/* ---------------------------------------------------------------------------------------------
 * Host-buffer entry point: one pass of the whole hot path (a2..a7) with HOST inputs and outputs.
 * The session owns device buffers sized for (max_edges, max_nodes), a compute stream and two copy
 * streams; each run copies the inputs host->device, runs graph_prepare, sh_fwd, tp_scatter_fwd,
 * tp_scatter_bwd, sh_bwd and force_reduce, copies the requested results device->host and synchronises.
 * The weights / out / grad_weights traffic is pipelined over contiguous receiver ranges (copy-in of range
 * k+1, compute of range k and copy-out of range k-1 overlap); results are bit-identical to the device
 * entry points on the same inputs.  Host buffers should be pinned for the overlap.  Any output pointer
 * may be NULL (skipped, and its copy is not made).  Inputs have the plan's storage dtype where
 * the device entry points do.  bytes_h2d / bytes_d2h (may be NULL) receive the bytes copied.
 * Preconditions, CHECKED on the host before anything is launched (one O(E) pass): every sender / receiver index lies
 * in [0, n_nodes) (else E3_ERR_INVALID_ARG) and receivers_h is ascending (else E3_ERR_UNSORTED).  On any failing
 * return the session's three streams have been synchronised: no copy still touches the caller's buffers.
 * -------------------------------------------------------------------------------------------*/
int e3_session_create(e3_session **session, const e3_plan *plan, int64_t max_edges, int32_t max_nodes);
int e3_session_destroy(e3_session *session);
int e3_session_run_host(e3_session *session, const float *vec_h, const void *feats_h, const void *weights_h,
                        const int32_t *senders_h, const int32_t *receivers_h, int64_t n_edges, int32_t n_nodes,
                        const float *grad_out_h, float *out_h, float *grad_feats_h, void *grad_weights_h,
                        float *grad_vec_h, float *forces_h, int64_t *bytes_h2d, int64_t *bytes_d2h);

/* ---------------------------------------------------------------------------------------------
 * NEXT-1: the radial network that GENERATES the weights.  PAPER.md L82 (fusing the message-passing
 * kernel is the authors' open item), L487-L491 (NequIP: num_rbf 8, swish, 64 hidden, 2 layers, polynomial envelope),
 * L539-L542 (MACE: num_rbf 16, polynomial envelope), L497 (5 A cutoff).  The paper prints no formula; readings R1-R4
 * (DESIGN.md): with r = |vec_e|, x = r / cutoff,
 *   f_k(r) = sqrt(2/cutoff) sin(k pi r / cutoff) / r * u(x),  k = 1..num_rbf,
 *   u(x) = 1 - (p+1)(p+2)/2 x^p + p(p+2) x^(p+1) - p(p+1)/2 x^(p+2)  (x < 1; 0 beyond),  p = envelope_p,
 *   w[e, :] = silu(silu(f W1) W2) W3,  silu(a) = a / (1 + exp(-a)),  W1[num_rbf, 64], W2[64, 64], W3[64, n_out], no biases,
 * and n_out = P*C so that w is exactly the `weights` operand of e3_tp_scatter_fwd/bwd of an E3_F32 plan.
 * The last layer (edges x 64 x n_out) runs on the tensor cores (tcgen05.mma kind::tf32, TMEM accumulators) as a 3xTF32
 * split product, accurate to fp32 rounding; the small layers run in fp32 on the CUDA cores.
 * e3_radial_create copies the (HOST, row-major, float) parameter matrices to the device and synchronises.
 * Limits: n_hidden == 64, num_rbf <= 16, n_out % 8 == 0 (else E3_ERR_UNSUPPORTED).
 * e3_radial_weights_fwd: weights[E, n_out] (float, device) from vec[E,3]; workspace >= e3_radial_workspace_bytes.
 * e3_radial_weights_bwd: given grad_weights[E, n_out] (float; the grad_weights output of e3_tp_scatter_bwd), computes
 *   dE/dr through the network and writes (accumulate == 0) or adds (accumulate != 0) dE/dr * vec/|vec| to grad_vec[E,3]
 *   (zero for a zero-length vector): adding it to the e3_sh_bwd result gives the full dE/dvec, which e3_force_reduce turns
 *   into forces.  Gradients with respect to W1, W2, W3 are not computed by this library.
 * Pointers 16-byte aligned; launches on `stream` only; deterministic.
 * -------------------------------------------------------------------------------------------*/
typedef struct e3_radial e3_radial;
int e3_radial_create(e3_radial **net, int num_rbf, int envelope_p, double cutoff, int n_hidden, int n_out,
                     const float *W1_h, const float *W2_h, const float *W3_h);
int e3_radial_destroy(e3_radial *net);
size_t e3_radial_workspace_bytes(const e3_radial *net, int64_t n_edges);
int e3_radial_weights_fwd(const e3_radial *net, const float *vec /*[E,3]*/, int64_t n_edges, float *weights /*[E,n_out]*/,
                          void *workspace, size_t workspace_bytes, e3_stream stream);
int e3_radial_weights_bwd(const e3_radial *net, const float *vec, int64_t n_edges, const float *grad_weights /*[E,n_out]*/,
                          float *grad_vec /*[E,3]*/, int accumulate, void *workspace, size_t workspace_bytes, e3_stream stream);

/* ---------------------------------------------------------------------------------------------
 * NEXT-2: second-order VJP, for Hessian rows and Hessian-label training.  PAPER.md L108-L126 (section 5.2),
 * Eq. 3 (H_ij = d2E/dr_i dr_j = -dF_i/dr_j) and Eq. 4 (rows of selected force components by reverse mode): a Hessian row is
 * the VJP of first-order VJP outputs.  With out = T(feats, sh, weights) (trilinear) and the first-order outputs
 * (grad_feats, grad_sh, grad_weights) of e3_tp_scatter_bwd for the cotangent grad_out, let
 *   S = <v_feats, grad_feats> + <v_sh, grad_sh> + <v_weights, grad_weights>.
 * e3_tp_scatter_vjp_vjp returns dS/d grad_out (gg_out [N,out_dim*C]), dS/d feats (g_feats [N,in_dim*C]), dS/d sh (g_sh
 * [E,sh_dim]) and dS/d weights (g_weights [E,P*C]), all float.  Any of v_feats / v_sh / v_weights may be NULL (= zero) and any
 * output may be NULL (not computed).  Built from the plan's forward and VJP kernels with one operand replaced by its cotangent
 * (exact, because T is trilinear); E3_F32 plans only (E3_ERR_UNSUPPORTED otherwise).  workspace >= e3_vjp_vjp_workspace_bytes.
 * e3_sh_bwd_bwd is the matching second derivative of the spherical harmonics: the VJP of (vec, grad_sh) -> grad_vec of
 * e3_sh_bwd for a cotangent u[E,3]:  g_sh[E,sh_dim] = J(vec) u  and  g_vec[E,3] = (sum_lm grad_sh[e,lm] Hess Y_lm(vec_e)) u_e
 * (zeros for a zero-length vector); either output may be NULL.
 * -------------------------------------------------------------------------------------------*/
size_t e3_vjp_vjp_workspace_bytes(const e3_plan *plan, int64_t n_edges, int32_t n_nodes);
int e3_tp_scatter_vjp_vjp(const e3_plan *plan, const void *feats, const void *sh, const void *weights, const int32_t *senders,
                          const int32_t *receivers, const int32_t *row_ptr, const int32_t *perm_s, const int32_t *col_ptr,
                          int64_t n_edges, int32_t n_nodes, const float *grad_out, const float *v_feats, const float *v_sh,
                          const float *v_weights, float *gg_out, float *g_feats, float *g_sh, float *g_weights,
                          void *workspace, size_t workspace_bytes, e3_stream stream);
int e3_sh_bwd_bwd(const e3_plan *plan, const float *vec, const float *grad_sh, const float *u, int64_t n_edges,
                  float *g_vec, float *g_sh, e3_stream stream);

/* ---------------------------------------------------------------------------------------------
 * NEXT-3: MACE's symmetric contraction at correlation order 2 on node features, the other operation the paper
 * routes to e3j.  PAPER.md L535 (`node_symmetry 2`), L536 (`correlation 2`), L545 (`symmetric_contraction_backend e3j`); no
 * formula is printed, so reading S1: for node n of species z = species[n] and channel u, every path k has the weight
 * weights[(z*n_paths + k)*C + u] and is
 *   linear     (i_in1, i_in2 = -1, i_out):  out[n, i_out, M, u] += W * feats[n, i_in1, M, u]              (same l and parity)
 *   quadratic  (i_in1, i_in2,      i_out):  out[n, i_out, M, u] += W * sum_{m1,m2} C[m1,m2,M] feats[n,i_in1,m1,u] feats[n,i_in2,m2,u]
 * with the real Clebsch-Gordan tensor C^{l1 l2 L} of reading A4 (triangle rule; parity p1*p2 = p_out; E3_ERR_BAD_PATH otherwise).
 * Layout A7 (blocks concatenated, index m*C + u); all multiplicities equal; float tensors on the device; species int32 in
 * [0, n_species) (values outside are clamped, never read out of bounds).  e3_symcon_bwd returns grad_feats [N,in_dim*C] and
 * grad_weights [n_species,n_paths,C] (either may be NULL) for grad_out = dL/d out; workspace >= e3_symcon_workspace_bytes is needed
 * for grad_weights.  Deterministic (every element is summed by one thread in a fixed order; grad_weights over node chunks -- their
 * number depends on n_nodes, C, the table sizes and the device type only -- in a fixed order).  A call that wants both gradients reads feats and
 * grad_out once (one combined kernel); its results are bit-identical to those of the single-gradient calls.  The kernels are specialised for the path table at creation (NVRTC; E3_SYMCON_JIT=0
 * keeps the table-driven fallback, which is also used beyond 6000 CG terms).  e3_symcon_create needs a device (the CG tensors come from the planner kernel) and synchronises.
 * -------------------------------------------------------------------------------------------*/
typedef struct e3_symcon e3_symcon;
typedef struct { int i_in1; int i_in2; int i_out; } e3_pair_path;
int e3_symcon_create(e3_symcon **sc, const e3_irrep *irreps_in, int n_in, const e3_irrep *irreps_out, int n_out,
                     const e3_pair_path *paths, int n_paths, int n_species);
int e3_symcon_destroy(e3_symcon *sc);
/* Build-time check (host only, no device needed): generates and compiles the specialised kernels of this path table for sm_100a; returns the
 * forward kernel's registers and spill bytes.  Same validation and status codes as e3_symcon_create. */
int e3_symcon_jit_check(const e3_irrep *irreps_in, int n_in, const e3_irrep *irreps_out, int n_out, const e3_pair_path *paths, int n_paths,
                        int *fwd_regs, int *fwd_spill);
int e3_symcon_dims(const e3_symcon *sc, int *in_dim, int *out_dim, int *n_paths, int *n_terms);
int e3_symcon_fwd(const e3_symcon *sc, const float *feats, const int32_t *species, const float *weights, int32_t n_nodes,
                  float *out, e3_stream stream);
size_t e3_symcon_workspace_bytes(const e3_symcon *sc, int32_t n_nodes);
int e3_symcon_bwd(const e3_symcon *sc, const float *feats, const int32_t *species, const float *weights, int32_t n_nodes,
                  const float *grad_out, float *grad_feats, float *grad_weights, void *workspace, size_t workspace_bytes,
                  e3_stream stream);

/* ---------------------------------------------------------------------------------------------
 * NEXT-4: neighbour list on the device.  PAPER.md L66 (the Graph class computes edge vectors from positions and
 * connectivity), L82 ("scale model deployment to larger systems"), L298 / L497 (5 A cutoff).  No formula is printed; reading N1
 * (DESIGN.md), evaluated in float32 with every operation rounded (no fused multiply-add) so that the edge set is unique:
 *   d_a = pos[r,a] - pos[s,a];   if box[a] > 0:  d_a = d_a - box[a] * rint(d_a / box[a])      (minimum image, reading A10)
 *   d2 = (d_x*d_x + d_y*d_y) + d_z*d_z;   edge s -> r  iff  s != r  and  d2 < cutoff*cutoff     (strict, reading A11)
 * Output, ordered by receiver with ties in ascending sender (A11), i.e. exactly what e3_tp_scatter_* expect:
 *   senders[E], receivers[E] (int32), vec[E,3] = d (float), row_ptr[N+1] (= the row_ptr of e3_graph_prepare).
 * pos [N,3] float on the device (any values; periodic axes are wrapped); box[3] on the HOST: edge length of a periodic axis, or 0
 * for an open axis; a periodic edge shorter than 2*cutoff is E3_ERR_UNSUPPORTED (a sender would have two images in range).
 * *n_edges (HOST) receives the edge count; if it exceeds max_edges (the capacity of senders / receivers / vec) nothing is written
 * to them and E3_ERR_WORKSPACE is returned with *n_edges set, so the caller can allocate and call again.  Uses a cell list
 * (integer atomics only); synchronises `stream` (the count is read back).  workspace >= e3_neighbor_workspace_bytes(n_nodes).
 * -------------------------------------------------------------------------------------------*/
size_t e3_neighbor_workspace_bytes(int32_t n_nodes);
int e3_neighbor_build(const float *pos /*[N,3]*/, int32_t n_nodes, const float *box /*[3], host*/, float cutoff, int64_t max_edges,
                      int32_t *senders, int32_t *receivers, float *vec /*[E,3]*/, int32_t *row_ptr /*[N+1]*/, int64_t *n_edges /*host*/,
                      void *workspace, size_t workspace_bytes, e3_stream stream);

/* ---------------------------------------------------------------------------------------------
 * NEXT-4 / SURVEY 8(e): receiver-range sharding of one graph over the GPUs of a node (HOST-side planning; all pointers are host
 * pointers, no device work).  PAPER.md L82; reading N2.  Rank k owns the atoms [bounds[k], bounds[k+1]) and all their
 * in-edges: boundary k is the receiver of edge floor(k*E/world) (n_nodes when that index is E), boundaries made non-decreasing,
 * so the ranks hold about equal edge counts.  receivers must be ascending (E3_ERR_UNSORTED).
 * e3_shard_localize describes the local problem of the owner of [lo, hi): its edge range [*e_lo, *e_hi), its halo (the senders
 * of its edges that it does not own, ascending global ids, *n_halo of them) and its edges with LOCAL node ids: owned atoms are
 * 0 .. hi-lo-1 in order, halo atoms follow in halo order.  halo, senders_local and receivers_local need room for *e_hi - *e_lo
 * entries; pass the three of them and n_halo as NULL to query the edge range first.  The local problem is an ordinary
 * e3_tp_scatter_fwd / _bwd call on hi-lo+n_halo nodes; paper_2605_22698_b200/sharded.py does the two exchanges with
 * torch.distributed (halo rows of feats in, halo rows of grad_feats back, added in rank order).
 * -------------------------------------------------------------------------------------------*/
int e3_shard_ranges(const int32_t *receivers_h, int64_t n_edges, int32_t n_nodes, int world, int32_t *bounds /*[world+1]*/);
int e3_shard_localize(const int32_t *senders_h, const int32_t *receivers_h, int64_t n_edges, int32_t n_nodes, int32_t lo, int32_t hi,
                      int64_t *e_lo, int64_t *e_hi, int32_t *halo, int32_t *n_halo, int32_t *senders_local, int32_t *receivers_local);

/* ---------------------------------------------------------------------------------------------
 * Graph preparation without any allocation (same operation, arguments and results as e3_graph_prepare: SURVEY 8(a) a3, readings
 * A11/A14/A15), for callers that cannot call cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses that forbid
 * it.  The scratch of e3_graph_prepare lives in a static device array of e3_graph_noalloc_capacity_bytes() = 32 MiB that every
 * GPU loading the library holds until the process exits; the call allocates and frees nothing (no cudaMalloc / cudaFree, no
 * allocating library routine).  Limit: e3_graph_workspace_bytes(n_edges, n_nodes) <= the capacity, i.e. n_edges + n_nodes <=
 * 8 388 600; beyond it E3_ERR_WORKSPACE is returned with the sizes in e3_last_error() and nothing is launched.
 * All pointers are device pointers owned by the caller (row_ptr[N+1], perm_s[E], col_ptr[N+1]); the device of `stream` must be
 * current.  validate != 0 synchronises `stream` as in e3_graph_prepare.
 * SHARING: every call on a device uses the same array.  Calls that overlap on the GPU (different streams, or threads that do not
 * order their calls) race on it and give undefined results; calls on one stream are ordered and safe.  The array keeps the last
 * call's contents; the call clears or overwrites everything it reads, so that is harmless.
 * -------------------------------------------------------------------------------------------*/
size_t e3_graph_noalloc_capacity_bytes(void);
int e3_graph_prepare_noalloc(const int32_t *senders, const int32_t *receivers, int64_t n_edges, int32_t n_nodes,
                             int32_t *row_ptr, int32_t *perm_s, int32_t *col_ptr, int validate, e3_stream stream);

#ifdef __cplusplus
}
#endif
#endif /* E3B200_H */
