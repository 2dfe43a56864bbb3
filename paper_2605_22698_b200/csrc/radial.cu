// NEXT-1: the radial network that GENERATES the per-edge weights w[e, p*C + u] from |vec_e|, and its VJP with
// respect to the edge vector (the extra force term).  PAPER.md L82 ("fusion of the message passing kernel" is the authors' open
// item), L487-L491 (NequIP: num_rbf 8, swish, 64 hidden, 2 layers, polynomial envelope), L539-L542 (MACE: num_rbf 16,
// polynomial envelope), L497 (5 A cutoff).  Formulas: readings R1-R4 of DESIGN.md (Bessel basis x polynomial envelope ->
// silu(f W1) -> silu(. W2) -> . W3).
//
// Kernels:
//   radial_hidden_kernel      vec -> r -> f[K] -> h1[64] -> h2[64]                (CUDA cores, fp32; 4.6 k FMA per edge)
//   radial_gemm_kernel        D[128 x 64 tile] = A[128 x Kt] * B[64 x Kt]^T on the 5th-generation tensor cores: tcgen05.mma
//                             kind::tf32 with TMEM accumulators, operands staged in shared memory in the canonical K-major
//                             no-swizzle core-matrix layout, 3xTF32 split (hi*hi + hi*lo + lo*hi) so that the result is fp32
//                             accurate (plain TF32 cannot meet the 1e-5 forward bar).  Used twice:
//                               forward   w[E, n_out]  = h2[E, 64] * W3[64, n_out]           (the dense edges x 64 x (P*C) product)
//                               backward  dh2[E, 64]   = dw[E, n_out] * W3[64, n_out]^T
//   radial_hidden_bwd_kernel  dh2 -> ... -> d r -> grad_vec += (dE/dr) vec/|vec|
// Gradients with respect to the network parameters (W1, W2, W3) are NOT built on the GPU (the oracle has them); this slice is
// what forces / MD need.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "e3_internal.h"

using namespace e3;

struct e3_radial {
    int K = 0, p = 6, H = 64, n_out = 0;
    double rc = 5.0;
    float *W1 = nullptr, *W2 = nullptr, *W2T = nullptr;        // [K,64], [64,64], transposed copy
    float *W3T_hi = nullptr, *W3T_lo = nullptr;                // [n_out,64]: W3^T split into TF32 high / low parts (B operand of the forward)
    float *W3_hi = nullptr, *W3_lo = nullptr;                  // [64,n_out]: W3 split (B operand of the backward)
};

namespace {

constexpr int kH = 64;          // hidden width
constexpr int kMaxRbf = 16;
constexpr int kTileM = 128, kTileN = 64, kTileK = 64;

__device__ __forceinline__ float silu_f(float a) { return a / (1.0f + expf(-a)); }
__device__ __forceinline__ float dsilu_f(float a) { const float s = 1.0f / (1.0f + expf(-a)); return s + a * s * (1.0f - s); }

// radial feature k (0-based) and its derivative with respect to r (readings R1, R2)
__device__ __forceinline__ void radial_feature(int k, float r, float rc, int p, float &f, float &dfdr)
{
    const float pi = 3.14159265358979323846f, nrm = sqrtf(2.0f / rc);
    const float a = (k + 1) * pi / rc;
    const float x = r / rc;
    float u = 0.0f, du = 0.0f;
    if (x < 1.0f) {
        const float ca = -0.5f * (p + 1) * (p + 2), cb = (float)p * (p + 2), cc = -0.5f * p * (p + 1);
        const float xp1 = powf(x, (float)(p - 1));         // x^(p-1)
        const float xp = xp1 * x;
        u = 1.0f + xp * (ca + x * (cb + x * cc));
        du = xp1 * (ca * p + x * (cb * (p + 1) + x * cc * (p + 2)));
    }
    float b, db;
    const float t = a * r;
    if (r > 0.0f) {
        float sn, cs;
        sincosf(t, &sn, &cs);
        b = nrm * sn / r;
        // a cos(t)/r - sin(t)/r^2 = (t cos t - sin t)/r^2; series for small t (cancellation)
        const float num = t < 0.3f ? t * t * t * (-1.0f / 3.0f + t * t * (1.0f / 30.0f - t * t * (1.0f / 840.0f))) : (t * cs - sn);
        db = nrm * num / (r * r);
    } else {
        b = nrm * a;
        db = 0.0f;
    }
    f = b * u;
    dfdr = db * u + b * du / rc;
}

// one warp per edge (grid-stride); lane owns hidden units `lane` and `lane + 32`
__global__ void __launch_bounds__(128) radial_hidden_kernel(const float *__restrict__ vec, long long E, int K, int p, float rc,
                                                            const float *__restrict__ W1, const float *__restrict__ W2, float *__restrict__ h2out)
{
    __shared__ float W1s[kMaxRbf * kH];
    __shared__ float W2s[kH * kH];
    for (int i = threadIdx.x; i < K * kH; i += blockDim.x) W1s[i] = W1[i];
    for (int i = threadIdx.x; i < kH * kH; i += blockDim.x) W2s[i] = W2[i];
    __syncthreads();
    const int lane = threadIdx.x & 31;
    const long long warp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long e = warp; e < E; e += nwarps) {
        const float vx = vec[3 * e], vy = vec[3 * e + 1], vz = vec[3 * e + 2];
        const float r = sqrtf(vx * vx + vy * vy + vz * vz);
        float f = 0.0f, dd;
        if (lane < K) radial_feature(lane, r, rc, p, f, dd);
        float a0 = 0.0f, a1 = 0.0f;
        for (int k = 0; k < K; ++k) {
            const float fk = __shfl_sync(0xffffffffu, f, k);
            a0 = fmaf(fk, W1s[k * kH + lane], a0);
            a1 = fmaf(fk, W1s[k * kH + lane + 32], a1);
        }
        const float h0 = silu_f(a0), h1 = silu_f(a1);
        float b0 = 0.0f, b1 = 0.0f;
#pragma unroll 8
        for (int i = 0; i < 32; ++i) {
            const float hi0 = __shfl_sync(0xffffffffu, h0, i), hi1 = __shfl_sync(0xffffffffu, h1, i);
            b0 = fmaf(hi0, W2s[i * kH + lane], b0);
            b1 = fmaf(hi0, W2s[i * kH + lane + 32], b1);
            b0 = fmaf(hi1, W2s[(i + 32) * kH + lane], b0);
            b1 = fmaf(hi1, W2s[(i + 32) * kH + lane + 32], b1);
        }
        h2out[e * kH + lane] = silu_f(b0);
        h2out[e * kH + lane + 32] = silu_f(b1);
    }
}

// backward of the hidden layers: dh2[E,64] -> d r -> grad_vec (+)= dE/dr * vec/|vec|
__global__ void __launch_bounds__(128) radial_hidden_bwd_kernel(const float *__restrict__ vec, long long E, int K, int p, float rc,
                                                                const float *__restrict__ W1, const float *__restrict__ W2, const float *__restrict__ W2T,
                                                                const float *__restrict__ dh2, float *__restrict__ gvec, int accumulate)
{
    __shared__ float W1s[kMaxRbf * kH];
    __shared__ float W2s[kH * kH];
    __shared__ float W2Ts[kH * kH];
    for (int i = threadIdx.x; i < K * kH; i += blockDim.x) W1s[i] = W1[i];
    for (int i = threadIdx.x; i < kH * kH; i += blockDim.x) { W2s[i] = W2[i]; W2Ts[i] = W2T[i]; }
    __syncthreads();
    const int lane = threadIdx.x & 31;
    const long long warp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long e = warp; e < E; e += nwarps) {
        const float vx = vec[3 * e], vy = vec[3 * e + 1], vz = vec[3 * e + 2];
        const float r = sqrtf(vx * vx + vy * vy + vz * vz);
        float f = 0.0f, dfdr = 0.0f;
        if (lane < K) radial_feature(lane, r, rc, p, f, dfdr);
        float a0 = 0.0f, a1 = 0.0f;
        for (int k = 0; k < K; ++k) {
            const float fk = __shfl_sync(0xffffffffu, f, k);
            a0 = fmaf(fk, W1s[k * kH + lane], a0);
            a1 = fmaf(fk, W1s[k * kH + lane + 32], a1);
        }
        const float h0 = silu_f(a0), h1 = silu_f(a1);
        float b0 = 0.0f, b1 = 0.0f;
#pragma unroll 8
        for (int i = 0; i < 32; ++i) {
            const float hi0 = __shfl_sync(0xffffffffu, h0, i), hi1 = __shfl_sync(0xffffffffu, h1, i);
            b0 = fmaf(hi0, W2s[i * kH + lane], b0);
            b1 = fmaf(hi0, W2s[i * kH + lane + 32], b1);
            b0 = fmaf(hi1, W2s[(i + 32) * kH + lane], b0);
            b1 = fmaf(hi1, W2s[(i + 32) * kH + lane + 32], b1);
        }
        // dL/da2 for units lane, lane + 32
        const float g20 = dh2[e * kH + lane] * dsilu_f(b0), g21 = dh2[e * kH + lane + 32] * dsilu_f(b1);
        // dL/dh1[i] = sum_j g2[j] W2[i][j]  (W2T[j][i] read contiguously over the lanes)
        float t0 = 0.0f, t1 = 0.0f;
#pragma unroll 8
        for (int j = 0; j < 32; ++j) {
            const float gj0 = __shfl_sync(0xffffffffu, g20, j), gj1 = __shfl_sync(0xffffffffu, g21, j);
            t0 = fmaf(gj0, W2Ts[j * kH + lane], t0);
            t1 = fmaf(gj0, W2Ts[j * kH + lane + 32], t1);
            t0 = fmaf(gj1, W2Ts[(j + 32) * kH + lane], t0);
            t1 = fmaf(gj1, W2Ts[(j + 32) * kH + lane + 32], t1);
        }
        const float g10 = t0 * dsilu_f(a0), g11 = t1 * dsilu_f(a1);
        // d f_k = sum_i g1[i] W1[k][i]; dr = sum_k d f_k * d f_k / d r   (fixed-order butterflies: deterministic)
        float dr = 0.0f;
        for (int k = 0; k < K; ++k) {
            float part = g10 * W1s[k * kH + lane] + g11 * W1s[k * kH + lane + 32];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
            const float dk = __shfl_sync(0xffffffffu, dfdr, k);
            dr = fmaf(part, dk, dr);
        }
        if (lane == 0) {
            const float inv = r > 0.0f ? 1.0f / r : 0.0f;
            const float gx = dr * vx * inv, gy = dr * vy * inv, gz = dr * vz * inv;
            if (accumulate) { gvec[3 * e] += gx; gvec[3 * e + 1] += gy; gvec[3 * e + 2] += gz; }
            else { gvec[3 * e] = gx; gvec[3 * e + 1] = gy; gvec[3 * e + 2] = gz; }
        }
    }
}

// split W3 into TF32 high / low parts, both as [64][n_out] and transposed [n_out][64]
__global__ void radial_split_w3_kernel(const float *__restrict__ W3, int n_out, float *__restrict__ hi, float *__restrict__ lo,
                                       float *__restrict__ thi, float *__restrict__ tlo)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= kH * n_out) return;
    const int j = i / n_out, n = i % n_out;
    const float v = W3[i];
    const float h = __uint_as_float(__float_as_uint(v) & 0xffffe000u);
    const float l = v - h;
    hi[i] = h; lo[i] = l;
    thi[n * kH + j] = h; tlo[n * kH + j] = l;
}

// ---------------------------------------------------------------------------------------------------------------------
// tcgen05 GEMM, 3xTF32:  D[m0 + 0..127, n0 + 0..63] = sum_k A[m, k] * B[n, k]   (A: M x Kt row-major (lda), B given as its TF32
// high and low parts, N x Kt row-major (ldb), D: M x N row-major (ldd)).  One CTA (4 warps) owns a 128-row tile and walks the
// N tiles (n_tiles) and, inside each, the K chunks of 64 (k_chunks).  Operand tiles live in shared memory in the canonical
// K-major no-swizzle layout: core matrices of 8 rows x 16 bytes, consecutive core matrices along K 128 bytes apart (LBO), groups
// of 8 rows 2048 bytes apart (SBO).  A is split into its TF32 high part (mantissa truncated to 10 bits, what the tensor core
// would read anyway) and the exact remainder; per K step of 8 the three products lo*hi, hi*lo, hi*hi accumulate into TMEM (fp32).
// ---------------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint64_t umma_desc(uint32_t smem_addr)
{
    uint64_t d = 0;
    d |= (uint64_t)((smem_addr >> 4) & 0x3fff);                 // start address
    d |= (uint64_t)((128u >> 4) & 0x3fff) << 16;                // leading-dimension byte offset: next core matrix along K
    d |= (uint64_t)((2048u >> 4) & 0x3fff) << 32;               // stride-dimension byte offset: next group of 8 rows
    d |= (uint64_t)1 << 46;                                     // descriptor version (sm_100)
    return d;                                                   // base offset 0, layout type 0 = no swizzle
}

__device__ __forceinline__ uint32_t canon_off(int row, int k)    // byte offset of element (row, k) of a [rows x 64] fp32 tile
{
    return (uint32_t)((row >> 3) * 2048 + (k >> 2) * 128 + (row & 7) * 16 + (k & 3) * 4);
}

__global__ void __launch_bounds__(128, 2) radial_gemm_kernel(const float *__restrict__ A, long long lda, const float *__restrict__ Bhi,
                                                             const float *__restrict__ Blo, long long ldb, float *__restrict__ D, long long ldd,
                                                             long long M, int N, int n_tiles, int k_chunks, long long Kt)
{
    extern __shared__ __align__(1024) unsigned char smem[];
    unsigned char *sAhi = smem, *sAlo = smem + 32768, *sBhi = smem + 65536, *sBlo = smem + 65536 + 16384;
    __shared__ __align__(8) unsigned long long mbar;
    __shared__ uint32_t tmem_base_s;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const long long m0 = (long long)blockIdx.x * kTileM;
    const uint32_t mbar_s = (uint32_t)__cvta_generic_to_shared(&mbar);
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 64;" :: "r"((uint32_t)__cvta_generic_to_shared(&tmem_base_s)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(mbar_s) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = tmem_base_s;
    // instruction descriptor: D fp32, A/B TF32, both K-major, N = 64, M = 128
    const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(kTileN >> 3) << 17) | ((uint32_t)(kTileM >> 4) << 24);
    const uint32_t sAhi_s = (uint32_t)__cvta_generic_to_shared(sAhi), sAlo_s = (uint32_t)__cvta_generic_to_shared(sAlo);
    const uint32_t sBhi_s = (uint32_t)__cvta_generic_to_shared(sBhi), sBlo_s = (uint32_t)__cvta_generic_to_shared(sBlo);
    uint32_t phase = 0;
    for (int nt = 0; nt < n_tiles; ++nt) {
        const int n0 = nt * kTileN;
        for (int kc = 0; kc < k_chunks; ++kc) {
            const long long k0 = (long long)kc * kTileK;
            // A chunk [128 x 64]: 2048 float4; thread t takes float4 (row = i / 16, quad = i % 16); a float4 is one core-matrix row
            if (nt == 0 || k_chunks > 1) {
                for (int i = tid; i < kTileM * 16; i += 128) {
                    const int row = i >> 4, q = i & 15;
                    float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (m0 + row < M && k0 + q * 4 + 4 <= Kt) v = *reinterpret_cast<const float4 *>(A + (m0 + row) * lda + k0 + q * 4);
                    float4 h, l;
                    h.x = __uint_as_float(__float_as_uint(v.x) & 0xffffe000u); l.x = v.x - h.x;
                    h.y = __uint_as_float(__float_as_uint(v.y) & 0xffffe000u); l.y = v.y - h.y;
                    h.z = __uint_as_float(__float_as_uint(v.z) & 0xffffe000u); l.z = v.z - h.z;
                    h.w = __uint_as_float(__float_as_uint(v.w) & 0xffffe000u); l.w = v.w - h.w;
                    const uint32_t off = canon_off(row, q * 4);
                    *reinterpret_cast<float4 *>(sAhi + off) = h;
                    *reinterpret_cast<float4 *>(sAlo + off) = l;
                }
            }
            // B chunk [64 x 64] (rows = output columns n0 + row, or zero beyond N)
            for (int i = tid; i < kTileN * 16; i += 128) {
                const int row = i >> 4, q = i & 15;
                float4 h = make_float4(0.f, 0.f, 0.f, 0.f), l = h;
                if (n0 + row < N && k0 + q * 4 + 4 <= Kt) {
                    h = *reinterpret_cast<const float4 *>(Bhi + (long long)(n0 + row) * ldb + k0 + q * 4);
                    l = *reinterpret_cast<const float4 *>(Blo + (long long)(n0 + row) * ldb + k0 + q * 4);
                }
                const uint32_t off = canon_off(row, q * 4);
                *reinterpret_cast<float4 *>(sBhi + off) = h;
                *reinterpret_cast<float4 *>(sBlo + off) = l;
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");       // generic-proxy stores -> visible to the tensor core (async proxy)
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            __syncthreads();
            if (tid == 0) {
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
                for (int ks = 0; ks < kTileK / 8; ++ks) {       // one MMA covers K = 8 (32 bytes = two core matrices): advance 256 bytes
                    const uint64_t ahi = umma_desc(sAhi_s + ks * 256), alo = umma_desc(sAlo_s + ks * 256);
                    const uint64_t bhi = umma_desc(sBhi_s + ks * 256), blo = umma_desc(sBlo_s + ks * 256);
                    const uint32_t acc0 = (kc > 0 || ks > 0) ? 1u : 0u;
                    asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n}"
                                 :: "r"(tmem), "l"(alo), "l"(bhi), "r"(idesc), "r"(acc0) : "memory");
                    asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n}"
                                 :: "r"(tmem), "l"(ahi), "l"(blo), "r"(idesc), "r"(1u) : "memory");
                    asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n}"
                                 :: "r"(tmem), "l"(ahi), "l"(bhi), "r"(idesc), "r"(1u) : "memory");
                }
                // arrives on the mbarrier when every MMA issued so far has completed (and has finished reading shared memory)
                asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(mbar_s) : "memory");
            }
            {
                asm volatile("{\n.reg .pred p;\nLAB_WAIT:\nmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n@p bra DONE;\nbra LAB_WAIT;\nDONE:\n}"
                             :: "r"(mbar_s), "r"(phase) : "memory");
                phase ^= 1u;
            }
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        }
        // epilogue: warp w reads TMEM lanes 32 w .. 32 w + 31 (= tile rows), 64 columns in two loads of 32
        const long long row = m0 + warp * 32 + lane;
#pragma unroll
        for (int c0 = 0; c0 < kTileN; c0 += 32) {
            uint32_t v[32];
            const uint32_t taddr = tmem + ((uint32_t)(warp * 32) << 16) + (uint32_t)c0;
            asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 "
                         "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
                         "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
                         : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
                           "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]),
                           "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]),
                           "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
                         : "r"(taddr) : "memory");
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
            if (row < M) {
                float *drow = D + row * ldd + n0 + c0;
                if (n0 + c0 + 32 <= N && (ldd & 3) == 0) {
#pragma unroll
                    for (int j = 0; j < 32; j += 4)
                        *reinterpret_cast<float4 *>(drow + j) = make_float4(__uint_as_float(v[j]), __uint_as_float(v[j + 1]), __uint_as_float(v[j + 2]), __uint_as_float(v[j + 3]));
                } else {
#pragma unroll
                    for (int j = 0; j < 32; ++j)
                        if (n0 + c0 + j < N) drow[j] = __uint_as_float(v[j]);
                }
            }
        }
        // the next tile overwrites TMEM and the B tiles: every warp must have drained its TMEM loads first
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    }
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 64;" :: "r"(tmem) : "memory");
}

constexpr int kGemmSmem = 65536 + 32768;

int launch_gemm(const float *A, long long lda, const float *Bhi, const float *Blo, long long ldb, float *D, long long ldd, long long M, int N,
                int n_tiles, int k_chunks, long long Kt, cudaStream_t st)
{
    static bool attr_set = false;
    if (!attr_set) {
        E3_CUDA_TRY(cudaFuncSetAttribute(radial_gemm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kGemmSmem));
        attr_set = true;
    }
    if (M <= 0) return E3_OK;
    const long long grid = (M + kTileM - 1) / kTileM;
    if (grid > 0x7fffffffLL) { set_error("radial gemm: grid too large"); return E3_ERR_UNSUPPORTED; }
    radial_gemm_kernel<<<(unsigned)grid, 128, kGemmSmem, st>>>(A, lda, Bhi, Blo, ldb, D, ldd, M, N, n_tiles, k_chunks, Kt);
    E3_CUDA_TRY(cudaGetLastError());
    return E3_OK;
}

}  // namespace

extern "C" int e3_radial_destroy(e3_radial *net)
{
    if (!net) return E3_OK;
    float *ptrs[] = { net->W1, net->W2, net->W2T, net->W3T_hi, net->W3T_lo, net->W3_hi, net->W3_lo };
    for (float *p : ptrs) if (p) cudaFree(p);
    delete net;
    return E3_OK;
}

extern "C" int e3_radial_create(e3_radial **net, int num_rbf, int envelope_p, double cutoff, int n_hidden, int n_out,
                                const float *W1_h, const float *W2_h, const float *W3_h)
{
    if (!net || !W1_h || !W2_h || !W3_h || num_rbf < 1 || n_out < 1 || !(cutoff > 0.0) || envelope_p < 2) {
        set_error("e3_radial_create: bad arguments");
        return E3_ERR_INVALID_ARG;
    }
    *net = nullptr;
    if (n_hidden != kH || num_rbf > kMaxRbf || (n_out % 8) != 0) {
        set_error("e3_radial_create: needs n_hidden == 64, num_rbf <= 16, n_out a multiple of 8 (got %d, %d, %d)", n_hidden, num_rbf, n_out);
        return E3_ERR_UNSUPPORTED;
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); set_error("e3_radial_create: no CUDA device (no CPU fallback)"); return E3_ERR_CUDA; }
    e3_radial *r = new (std::nothrow) e3_radial();
    if (!r) { set_error("out of host memory"); return E3_ERR_INVALID_ARG; }
    r->K = num_rbf; r->p = envelope_p; r->rc = cutoff; r->n_out = n_out;
    std::vector<float> w2t((size_t)kH * kH);
    for (int i = 0; i < kH; ++i) for (int j = 0; j < kH; ++j) w2t[(size_t)j * kH + i] = W2_h[(size_t)i * kH + j];
    const size_t n3 = (size_t)kH * n_out * sizeof(float);
    float *w3_tmp = nullptr;
    cudaError_t e = cudaMalloc(&r->W1, sizeof(float) * num_rbf * kH);
    if (e == cudaSuccess) e = cudaMalloc(&r->W2, sizeof(float) * kH * kH);
    if (e == cudaSuccess) e = cudaMalloc(&r->W2T, sizeof(float) * kH * kH);
    if (e == cudaSuccess) e = cudaMalloc(&r->W3T_hi, n3);
    if (e == cudaSuccess) e = cudaMalloc(&r->W3T_lo, n3);
    if (e == cudaSuccess) e = cudaMalloc(&r->W3_hi, n3);
    if (e == cudaSuccess) e = cudaMalloc(&r->W3_lo, n3);
    if (e == cudaSuccess) e = cudaMalloc(&w3_tmp, n3);
    if (e == cudaSuccess) e = cudaMemcpy(r->W1, W1_h, sizeof(float) * num_rbf * kH, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(r->W2, W2_h, sizeof(float) * kH * kH, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(r->W2T, w2t.data(), sizeof(float) * kH * kH, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(w3_tmp, W3_h, n3, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        radial_split_w3_kernel<<<(kH * n_out + 255) / 256, 256>>>(w3_tmp, n_out, r->W3_hi, r->W3_lo, r->W3T_hi, r->W3T_lo);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (w3_tmp) cudaFree(w3_tmp);
    if (e != cudaSuccess) { e3_radial_destroy(r); return cuda_fail(e, "e3_radial_create"); }
    *net = r;
    return E3_OK;
}

extern "C" size_t e3_radial_workspace_bytes(const e3_radial *net, int64_t n_edges)
{
    if (!net || n_edges < 0) return 0;
    return (size_t)n_edges * kH * sizeof(float) + 256;       // h2 (forward) or dh2 (backward), [E,64] fp32
}

extern "C" int e3_radial_weights_fwd(const e3_radial *net, const float *vec, int64_t n_edges, float *weights, void *workspace,
                                     size_t workspace_bytes, e3_stream stream)
{
    if (!net || n_edges < 0 || (n_edges > 0 && (!vec || !weights))) { set_error("e3_radial_weights_fwd: bad arguments"); return E3_ERR_INVALID_ARG; }
    if (n_edges == 0) return E3_OK;
    if (!workspace || workspace_bytes < e3_radial_workspace_bytes(net, n_edges)) { set_error("e3_radial_weights_fwd: workspace too small"); return E3_ERR_WORKSPACE; }
    if ((reinterpret_cast<uintptr_t>(weights) & 15u) || (reinterpret_cast<uintptr_t>(workspace) & 15u)) { set_error("e3_radial_weights_fwd: pointers must be 16-byte aligned"); return E3_ERR_INVALID_ARG; }
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    float *h2 = reinterpret_cast<float *>(workspace);
    const long long blocks = std::min<long long>((n_edges + 3) / 4, 148LL * 16);
    radial_hidden_kernel<<<(unsigned)blocks, 128, 0, st>>>(vec, n_edges, net->K, net->p, (float)net->rc, net->W1, net->W2, h2);
    E3_CUDA_TRY(cudaGetLastError());
    return launch_gemm(h2, kH, net->W3T_hi, net->W3T_lo, kH, weights, net->n_out, n_edges, net->n_out, (net->n_out + kTileN - 1) / kTileN, 1, kH, st);
}

extern "C" int e3_radial_weights_bwd(const e3_radial *net, const float *vec, int64_t n_edges, const float *grad_weights, float *grad_vec,
                                     int accumulate, void *workspace, size_t workspace_bytes, e3_stream stream)
{
    if (!net || n_edges < 0 || (n_edges > 0 && (!vec || !grad_weights || !grad_vec))) { set_error("e3_radial_weights_bwd: bad arguments"); return E3_ERR_INVALID_ARG; }
    if (n_edges == 0) return E3_OK;
    if (!workspace || workspace_bytes < e3_radial_workspace_bytes(net, n_edges)) { set_error("e3_radial_weights_bwd: workspace too small"); return E3_ERR_WORKSPACE; }
    if ((reinterpret_cast<uintptr_t>(grad_weights) & 15u) || (reinterpret_cast<uintptr_t>(workspace) & 15u)) { set_error("e3_radial_weights_bwd: pointers must be 16-byte aligned"); return E3_ERR_INVALID_ARG; }
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    float *dh2 = reinterpret_cast<float *>(workspace);
    // dh2[E,64] = dw[E,n_out] * W3[64,n_out]^T : A = dw (K = n_out), B = W3 rows (K-major), one N tile, n_out / 64 K chunks
    int rc = launch_gemm(grad_weights, net->n_out, net->W3_hi, net->W3_lo, net->n_out, dh2, kH, n_edges, kH, 1, (net->n_out + kTileK - 1) / kTileK, net->n_out, st);
    if (rc != E3_OK) return rc;
    const long long blocks = std::min<long long>((n_edges + 3) / 4, 148LL * 16);
    radial_hidden_bwd_kernel<<<(unsigned)blocks, 128, 0, st>>>(vec, n_edges, net->K, net->p, (float)net->rc, net->W1, net->W2, net->W2T, dh2, grad_vec, accumulate);
    E3_CUDA_TRY(cudaGetLastError());
    return E3_OK;
}
