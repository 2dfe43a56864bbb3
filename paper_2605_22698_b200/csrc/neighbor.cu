// NEXT-4 (the Graph class computes edge vectors from positions and connectivity; L82 "scale model
// deployment to larger systems"; L298 / L497: 5 A cutoff): neighbour list built on the device with a cell list.
//
// Reading N1 fixes WHICH edges exist, in float32 with every operation rounded (no fused multiply-add), so that the
// integer output is unique and bit-comparable with the brute-force oracle:
//     d_a = pos[r,a] - pos[s,a];   box_a > 0:  d_a = d_a - box_a * rint(d_a / box_a)
//     d2  = (d_x*d_x + d_y*d_y) + d_z*d_z;   edge s -> r  iff  s != r  and  d2 < cutoff*cutoff;   vec = d
// The cell list only narrows the CANDIDATES (cells are 1.0001 x cutoff wide or wider, so rounding in the cell assignment can
// never hide a pair that passes the test); the test itself is the formula above, evaluated with _rn intrinsics.
//
// Pipeline (integer atomics only; every float result is computed by one thread):
//   cell_count -> scan -> cell_fill            atoms bucketed by cell (order inside a cell is arbitrary and does not matter)
//   nb_count   -> scan                         one warp per receiver: degree over the <= 27 neighbouring cells -> row_ptr
//   nb_fill                                    one warp per receiver: accepted senders (unsorted, parked in `receivers`),
//                                              rank sort by sender id (ids are unique per receiver: one image at most),
//                                              senders / vec / receivers written in (receiver, sender) order (reading A11)
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>

#include "e3_internal.h"

using namespace e3;

namespace {

struct Grid {
    float box[3];      // periodic length, 0 = open
    float org[3];      // open dims: lower corner
    float inv_w[3];    // 1 / cell width
    int nc[3];
};

__device__ __forceinline__ int cell_coord(float x, const Grid &g, int a)
{
    float t;
    if (g.box[a] > 0.f) {
        const float f = x / g.box[a];
        t = (f - floorf(f)) * (float)g.nc[a];
    } else {
        t = (x - g.org[a]) * g.inv_w[a];
    }
    int c = (int)floorf(t);
    return c < 0 ? 0 : (c >= g.nc[a] ? g.nc[a] - 1 : c);
}

// order-preserving float <-> int map for atomicMin / atomicMax
__device__ __forceinline__ int f2ord(float f) { const int i = __float_as_int(f); return i >= 0 ? i : i ^ 0x7fffffff; }
__host__ __device__ __forceinline__ float ord2f(int i)
{
    const int j = i >= 0 ? i : i ^ 0x7fffffff;
#ifdef __CUDA_ARCH__
    return __int_as_float(j);
#else
    float f;
    memcpy(&f, &j, 4);
    return f;
#endif
}

__global__ void nb_bounds_kernel(const float *__restrict__ pos, int32_t N, int *__restrict__ mm /*[6]: min xyz, max xyz (ordered ints)*/)
{
    const int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    int lo[3], hi[3];
    for (int a = 0; a < 3; ++a) {
        const int v = i < N ? f2ord(pos[(size_t)i * 3 + a]) : 0;
        lo[a] = i < N ? v : 0x7fffffff;
        hi[a] = i < N ? v : (int)0x80000000;
    }
    for (int a = 0; a < 3; ++a) {
        for (int o = 16; o > 0; o >>= 1) {
            lo[a] = min(lo[a], __shfl_xor_sync(0xffffffffu, lo[a], o));
            hi[a] = max(hi[a], __shfl_xor_sync(0xffffffffu, hi[a], o));
        }
        if ((threadIdx.x & 31) == 0) { atomicMin(&mm[a], lo[a]); atomicMax(&mm[3 + a], hi[a]); }
    }
}

__global__ void nb_cell_count_kernel(const float *__restrict__ pos, int32_t N, Grid g, int32_t *__restrict__ cell_of, int32_t *__restrict__ cell_ptr)
{
    const int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int cx = cell_coord(pos[(size_t)i * 3 + 0], g, 0), cy = cell_coord(pos[(size_t)i * 3 + 1], g, 1), cz = cell_coord(pos[(size_t)i * 3 + 2], g, 2);
    const int c = (cx * g.nc[1] + cy) * g.nc[2] + cz;
    cell_of[i] = c;
    atomicAdd(&cell_ptr[c + 1], 1);
}

__global__ void nb_cell_fill_kernel(const int32_t *__restrict__ cell_of, int32_t N, int32_t *__restrict__ cursor, int32_t *__restrict__ cell_atoms)
{
    const int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) cell_atoms[atomicAdd(&cursor[cell_of[i]], 1)] = i;
}

// reading N1, every operation rounded to float32
__device__ __forceinline__ float min_image(float d, float box)
{
    return box > 0.f ? __fsub_rn(d, __fmul_rn(box, rintf(__fdiv_rn(d, box)))) : d;
}
__device__ __forceinline__ bool edge_test(const float pr[3], const float *__restrict__ ps, const Grid &g, float rc2, float d[3])
{
    d[0] = min_image(__fsub_rn(pr[0], ps[0]), g.box[0]);
    d[1] = min_image(__fsub_rn(pr[1], ps[1]), g.box[1]);
    d[2] = min_image(__fsub_rn(pr[2], ps[2]), g.box[2]);
    const float d2 = __fadd_rn(__fadd_rn(__fmul_rn(d[0], d[0]), __fmul_rn(d[1], d[1])), __fmul_rn(d[2], d[2]));
    return d2 < rc2;
}

// neighbouring cell coordinates along one axis without repeats: all of them when the axis has <= 3 cells
__device__ __forceinline__ int axis_cells(int c, int nc, bool periodic, int out[3])
{
    if (nc <= 3) { for (int k = 0; k < nc; ++k) out[k] = k; return nc; }
    int n = 0;
    for (int o = -1; o <= 1; ++o) {
        int k = c + o;
        if (periodic) k = k < 0 ? k + nc : (k >= nc ? k - nc : k);
        else if (k < 0 || k >= nc) continue;
        out[n++] = k;
    }
    return n;
}

// FILL = false: deg[r + 1] = degree.  FILL = true: the receiver's edges, sorted by sender.
template <bool FILL>
__global__ void __launch_bounds__(256) nb_edges_kernel(const float *__restrict__ pos, int32_t N, Grid g, float rc2, const int32_t *__restrict__ cell_of,
                                                       const int32_t *__restrict__ cell_ptr, const int32_t *__restrict__ cell_atoms,
                                                       int32_t *__restrict__ row_ptr, int32_t *__restrict__ senders, int32_t *receivers, float *__restrict__ vec)
{
    const int32_t r = (int32_t)(((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5);
    if (r >= N) return;
    const int lane = threadIdx.x & 31;
    const float pr[3] = { pos[(size_t)r * 3], pos[(size_t)r * 3 + 1], pos[(size_t)r * 3 + 2] };
    const int c = cell_of[r];
    const int cz = c % g.nc[2], cy = (c / g.nc[2]) % g.nc[1], cx = c / (g.nc[2] * g.nc[1]);
    int xs[3], ys[3], zs[3];
    const int nx = axis_cells(cx, g.nc[0], g.box[0] > 0.f, xs), ny = axis_cells(cy, g.nc[1], g.box[1] > 0.f, ys), nz = axis_cells(cz, g.nc[2], g.box[2] > 0.f, zs);
    const int32_t base = FILL ? row_ptr[r] : 0;
    int32_t count = 0;
    for (int ix = 0; ix < nx; ++ix)
        for (int iy = 0; iy < ny; ++iy)
            for (int iz = 0; iz < nz; ++iz) {
                const int cc = (xs[ix] * g.nc[1] + ys[iy]) * g.nc[2] + zs[iz];
                const int32_t a = cell_ptr[cc], b = cell_ptr[cc + 1];
                for (int32_t j0 = a; j0 < b; j0 += 32) {
                    const int32_t j = j0 + lane;
                    int32_t s = -1;
                    bool ok = false;
                    if (j < b) {
                        s = cell_atoms[j];
                        float d[3];
                        ok = s != r && edge_test(pr, pos + (size_t)s * 3, g, rc2, d);
                    }
                    const unsigned m = __ballot_sync(0xffffffffu, ok);
                    if (FILL && ok) receivers[base + count + __popc(m & ((1u << lane) - 1))] = s;      // unsorted, parked in `receivers`
                    count += __popc(m);
                }
            }
    if (!FILL) {
        if (lane == 0) row_ptr[r + 1] = count;
        return;
    }
    __syncwarp();
    // rank sort: sender ids of one receiver are distinct (a periodic box edge is at least twice the cutoff)
    for (int32_t i = lane; i < count; i += 32) {
        const int32_t s = receivers[base + i];
        int32_t rank = 0;
        for (int32_t j = 0; j < count; ++j) rank += receivers[base + j] < s;
        float d[3];
        edge_test(pr, pos + (size_t)s * 3, g, rc2, d);
        senders[base + rank] = s;
        vec[(size_t)(base + rank) * 3 + 0] = d[0];
        vec[(size_t)(base + rank) * 3 + 1] = d[1];
        vec[(size_t)(base + rank) * 3 + 2] = d[2];
    }
    __syncwarp();
    for (int32_t i = lane; i < count; i += 32) receivers[base + i] = r;
}

inline size_t up256(size_t b) { return (b + 255) / 256 * 256; }
constexpr int kMaxCellsPerAxis = 1024;

}  // namespace

// workspace: [0,256) bounds; cell_of[N]; cell_ptr[max_cells+1]; cursor[max_cells+1]; cell_atoms[N]
static size_t max_cells(int32_t N) { return (size_t)4 * (size_t)N + 64; }

extern "C" size_t e3_neighbor_workspace_bytes(int32_t n_nodes)
{
    if (n_nodes < 0) return 0;
    return 256 + up256(sizeof(int32_t) * (size_t)n_nodes) * 2 + up256(sizeof(int32_t) * (max_cells(n_nodes) + 2)) * 2;
}

extern "C" int e3_neighbor_build(const float *pos, int32_t n_nodes, const float *box, float cutoff, int64_t max_edges, int32_t *senders,
                                 int32_t *receivers, float *vec, int32_t *row_ptr, int64_t *n_edges, void *workspace, size_t workspace_bytes,
                                 e3_stream stream)
{
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    if (n_nodes < 0 || max_edges < 0 || !box || !row_ptr || !n_edges || !(cutoff > 0.f) || (n_nodes > 0 && !pos) ||
        (max_edges > 0 && (!senders || !receivers || !vec))) {
        set_error("e3_neighbor_build: bad arguments");
        return E3_ERR_INVALID_ARG;
    }
    *n_edges = 0;
    for (int a = 0; a < 3; ++a) {
        if (box[a] < 0.f || !(box[a] == box[a])) { set_error("e3_neighbor_build: box[%d] is negative or NaN", a); return E3_ERR_INVALID_ARG; }
        if (box[a] > 0.f && box[a] < 2.f * cutoff) {
            set_error("e3_neighbor_build: periodic box edge %g is shorter than twice the cutoff %g (a sender would have two images in range)", box[a], cutoff);
            return E3_ERR_UNSUPPORTED;
        }
    }
    if (!workspace || workspace_bytes < e3_neighbor_workspace_bytes(n_nodes)) { set_error("e3_neighbor_build: workspace too small"); return E3_ERR_WORKSPACE; }
    if (n_nodes == 0) { E3_CUDA_TRY(cudaMemsetAsync(row_ptr, 0, sizeof(int32_t), st)); return E3_OK; }
    char *wp = (char *)workspace;
    int *mm = (int *)wp; wp += 256;
    int32_t *cell_of = (int32_t *)wp; wp += up256(sizeof(int32_t) * (size_t)n_nodes);
    int32_t *cell_atoms = (int32_t *)wp; wp += up256(sizeof(int32_t) * (size_t)n_nodes);
    int32_t *cell_ptr = (int32_t *)wp; wp += up256(sizeof(int32_t) * (max_cells(n_nodes) + 2));
    int32_t *cursor = (int32_t *)wp;
    const unsigned tb = 256, gn = (unsigned)((n_nodes + tb - 1) / tb);
    Grid g;
    const float width = cutoff * 1.0001f;       // candidate cells are wider than the cutoff: cell-assignment rounding cannot hide a pair
    bool open = false;
    for (int a = 0; a < 3; ++a) { g.box[a] = box[a]; g.org[a] = 0.f; g.inv_w[a] = 0.f; g.nc[a] = 1; open = open || box[a] == 0.f; }
    float ext[3] = { 0.f, 0.f, 0.f };
    if (open) {                                  // bounding box of the atoms along the open axes
        const int init[6] = { 0x7fffffff, 0x7fffffff, 0x7fffffff, (int)0x80000000, (int)0x80000000, (int)0x80000000 };
        E3_CUDA_TRY(cudaMemcpyAsync(mm, init, sizeof(init), cudaMemcpyHostToDevice, st));
        nb_bounds_kernel<<<gn, tb, 0, st>>>(pos, n_nodes, mm);
        int h[6];
        E3_CUDA_TRY(cudaMemcpyAsync(h, mm, sizeof(h), cudaMemcpyDeviceToHost, st));
        E3_CUDA_TRY(cudaStreamSynchronize(st));
        for (int a = 0; a < 3; ++a) {
            const float lo = ord2f(h[a]), hi = ord2f(h[3 + a]);
            if (!(lo == lo) || !(hi == hi) || std::isinf(lo) || std::isinf(hi)) { set_error("e3_neighbor_build: positions contain NaN or infinity"); return E3_ERR_INVALID_ARG; }
            if (box[a] == 0.f) { g.org[a] = lo; ext[a] = hi - lo; }
        }
    }
    for (int a = 0; a < 3; ++a) {
        const float len = box[a] > 0.f ? box[a] : ext[a];
        int nc = (int)std::floor(len / width);
        if (box[a] == 0.f) nc += 1;              // open axis: cells of exactly `width` from the lower corner
        g.nc[a] = std::max(1, std::min(kMaxCellsPerAxis, nc));
    }
    while ((size_t)g.nc[0] * g.nc[1] * g.nc[2] > max_cells(n_nodes)) {       // sparse systems: widen the cells of the longest axis
        int a = 0;
        for (int k = 1; k < 3; ++k) if (g.nc[k] > g.nc[a]) a = k;
        g.nc[a] = (g.nc[a] + 1) / 2;
    }
    for (int a = 0; a < 3; ++a)
        if (box[a] == 0.f) {
            // nc cells must cover [org, org + ext]: width_a = max(width, ext / nc * (1 + 1e-6))
            const float wa = std::max(width, ext[a] / (float)g.nc[a] * 1.000001f);
            g.inv_w[a] = 1.f / wa;
        }
    const int32_t ncell = g.nc[0] * g.nc[1] * g.nc[2];
    E3_CUDA_TRY(cudaMemsetAsync(cell_ptr, 0, sizeof(int32_t) * ((size_t)ncell + 1), st));
    nb_cell_count_kernel<<<gn, tb, 0, st>>>(pos, n_nodes, g, cell_of, cell_ptr);
    int rc = launch_scan_i32(cell_ptr, ncell + 1, cursor, st);
    if (rc != E3_OK) return rc;
    nb_cell_fill_kernel<<<gn, tb, 0, st>>>(cell_of, n_nodes, cursor, cell_atoms);
    const float rc2 = cutoff * cutoff;           // host float multiply: one rounding, like the oracle's
    const unsigned gw = (unsigned)(((int64_t)n_nodes * 32 + tb - 1) / tb);
    E3_CUDA_TRY(cudaMemsetAsync(row_ptr, 0, sizeof(int32_t), st));
    nb_edges_kernel<false><<<gw, tb, 0, st>>>(pos, n_nodes, g, rc2, cell_of, cell_ptr, cell_atoms, row_ptr, nullptr, nullptr, nullptr);
    // degrees of up to 2^31 edges in total: the scan is int32, the total is checked on the host
    rc = launch_scan_i32(row_ptr, n_nodes + 1, cursor /*unused output*/, st);
    if (rc != E3_OK) return rc;
    int32_t total = 0;
    E3_CUDA_TRY(cudaMemcpyAsync(&total, row_ptr + n_nodes, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    E3_CUDA_TRY(cudaStreamSynchronize(st));
    E3_CUDA_TRY(cudaGetLastError());
    if (total < 0) { set_error("e3_neighbor_build: more than 2^31 - 1 edges"); return E3_ERR_UNSUPPORTED; }
    *n_edges = total;
    if ((int64_t)total > max_edges) {
        set_error("e3_neighbor_build: %d edges do not fit max_edges = %lld (n_edges holds the count; call again with larger buffers)", total, (long long)max_edges);
        return E3_ERR_WORKSPACE;
    }
    if (total > 0) nb_edges_kernel<true><<<gw, tb, 0, st>>>(pos, n_nodes, g, rc2, cell_of, cell_ptr, cell_atoms, row_ptr, senders, receivers, vec);
    E3_CUDA_TRY(cudaGetLastError());
    return E3_OK;
}
