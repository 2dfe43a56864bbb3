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
#include <cstdlib>
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

// Hidden layers, forward and (BWD) their VJP.  A warp processes EIGHT edges per pass; a lane owns hidden units `lane` and `lane + 32`
// of all eight.  The activations of the previous layer sit transposed in a per-warp shared-memory buffer [unit][edge], so two broadcast
// 16-byte loads serve sixteen FMAs (two units x eight edges) beside the two weight loads: 4 LDS per 16 FMA.  (One edge per warp: 2 LDS +
// 2 SHFL per 2 FMA, 87 % of the LSU pipe; four edges per pass: 3 LDS per 8 FMA, still LSU-bound at 54 %, profiles/r02c_radial_cfg4_full.md.)
constexpr int kEP = 8;          // edges per warp pass

template <bool BWD>
__global__ void __launch_bounds__(128) radial_hidden_kernel(const float *__restrict__ vec, long long E, int K, int p, float rc,
                                                            const float *__restrict__ W1, const float *__restrict__ W2, const float *__restrict__ W2T,
                                                            float *__restrict__ h2out, const float *__restrict__ dh2, float *__restrict__ gvec, int accumulate)
{
    extern __shared__ __align__(16) float hsm[];
    float *W1s = hsm;                                   // [K][64]
    float *W2s = W1s + kMaxRbf * kH;                    // [64][64]
    float *W2Ts = W2s + kH * kH;                        // [64][64] transposed (BWD only)
    float *W1Ts = W2Ts + (BWD ? kH * kH : 0);           // [64][4][4] (BWD only): W1[k = kk + 4 c][unit] at [unit][kk][c]
    float *wbuf = W1Ts + (BWD ? kH * kMaxRbf : 0);      // per warp: act[64][8] + feat[16][8]
    for (int i = threadIdx.x; i < kMaxRbf * kH; i += blockDim.x) W1s[i] = i < K * kH ? W1[i] : 0.0f;
    for (int i = threadIdx.x; i < kH * kH; i += blockDim.x) { W2s[i] = W2[i]; if (BWD) W2Ts[i] = W2T[i]; }
    if (BWD)
        for (int i = threadIdx.x; i < kH * kMaxRbf; i += blockDim.x) {
            const int u = i / kMaxRbf, kq = (i % kMaxRbf) >> 2, c = i & 3, k = kq + 4 * c;
            W1Ts[i] = k < K ? W1[k * kH + u] : 0.0f;
        }
    __syncthreads();
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    float *act = wbuf + wib * (kH * kEP + kMaxRbf * kEP), *feat = act + kH * kEP;
    const long long warp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
    const int el = lane >> 2, kk = lane & 3;            // this lane evaluates radial features kk, kk + 4, kk + 8, kk + 12 of edge el
    for (long long e0 = warp * kEP; e0 < E; e0 += nwarps * kEP) {
        const long long em = e0 + el < E ? e0 + el : E - 1;
        const float vx = vec[3 * em], vy = vec[3 * em + 1], vz = vec[3 * em + 2];
        const float r = sqrtf(vx * vx + vy * vy + vz * vz);
        float f[4] = { 0.f, 0.f, 0.f, 0.f }, d[4] = { 0.f, 0.f, 0.f, 0.f };
#pragma unroll
        for (int c = 0; c < 4; ++c)
            if (kk + 4 * c < K) radial_feature(kk + 4 * c, r, rc, p, f[c], d[c]);
        __syncwarp();
#pragma unroll
        for (int c = 0; c < 4; ++c) feat[(kk + 4 * c) * kEP + el] = f[c];
        __syncwarp();
        float a1[2][kEP] = {};
        for (int k = 0; k < K; ++k) {
            const float4 fa = *reinterpret_cast<const float4 *>(feat + k * kEP), fb = *reinterpret_cast<const float4 *>(feat + k * kEP + 4);
            const float fk[kEP] = { fa.x, fa.y, fa.z, fa.w, fb.x, fb.y, fb.z, fb.w };
            const float w0 = W1s[k * kH + lane], w1 = W1s[k * kH + lane + 32];
#pragma unroll
            for (int q = 0; q < kEP; ++q) { a1[0][q] = fmaf(fk[q], w0, a1[0][q]); a1[1][q] = fmaf(fk[q], w1, a1[1][q]); }
        }
        auto put = [&](int unit, const float (&v)[kEP]) {
            *reinterpret_cast<float4 *>(act + unit * kEP) = make_float4(v[0], v[1], v[2], v[3]);
            *reinterpret_cast<float4 *>(act + unit * kEP + 4) = make_float4(v[4], v[5], v[6], v[7]);
        };
        {
            float s0[kEP], s1[kEP];
#pragma unroll
            for (int q = 0; q < kEP; ++q) { s0[q] = silu_f(a1[0][q]); s1[q] = silu_f(a1[1][q]); }
            put(lane, s0); put(lane + 32, s1);
        }
        __syncwarp();
        // out[u][q] = sum_i act[i][q] * Wm[i][u] for u = lane, lane + 32 (Wm = W2 forward, W2^T for the VJP)
        auto layer = [&](const float *Wm, float (&o)[2][kEP]) {
#pragma unroll
            for (int q = 0; q < kEP; ++q) { o[0][q] = 0.f; o[1][q] = 0.f; }
#pragma unroll 8
            for (int i = 0; i < kH; ++i) {
                const float4 ha = *reinterpret_cast<const float4 *>(act + i * kEP), hb = *reinterpret_cast<const float4 *>(act + i * kEP + 4);
                const float h[kEP] = { ha.x, ha.y, ha.z, ha.w, hb.x, hb.y, hb.z, hb.w };
                const float w0 = Wm[i * kH + lane], w1 = Wm[i * kH + lane + 32];
#pragma unroll
                for (int q = 0; q < kEP; ++q) { o[0][q] = fmaf(h[q], w0, o[0][q]); o[1][q] = fmaf(h[q], w1, o[1][q]); }
            }
        };
        float a2[2][kEP];
        layer(W2s, a2);
        if (!BWD) {
#pragma unroll
            for (int q = 0; q < kEP; ++q)
                if (e0 + q < E) {      // h2 split into its TF32 high part and the exact remainder: the B operand of the output-layer GEMM
                    const float v0 = silu_f(a2[0][q]), v1 = silu_f(a2[1][q]);
                    const float h0 = __uint_as_float(__float_as_uint(v0) & 0xffffe000u), h1 = __uint_as_float(__float_as_uint(v1) & 0xffffe000u);
                    h2out[(e0 + q) * kH + lane] = h0; h2out[(e0 + q) * kH + lane + 32] = h1;
                    h2out[(E + e0 + q) * kH + lane] = v0 - h0; h2out[(E + e0 + q) * kH + lane + 32] = v1 - h1;
                }
            continue;
        }
        // ---- VJP: dL/da2 -> dL/dh1 -> dL/da1 -> d f -> d r
        {
            float g0[kEP], g1[kEP];
#pragma unroll
            for (int q = 0; q < kEP; ++q) {
                const long long eq = e0 + q < E ? e0 + q : E - 1;
                g0[q] = dh2[eq * kH + lane] * dsilu_f(a2[0][q]);
                g1[q] = dh2[eq * kH + lane + 32] * dsilu_f(a2[1][q]);
            }
            __syncwarp();
            put(lane, g0); put(lane + 32, g1);
        }
        __syncwarp();
        float t[2][kEP];
        layer(W2Ts, t);                                  // dL/dh1[i] = sum_j g2[j] W2[i][j]; W2T[j][i] is contiguous over the lanes
        __syncwarp();
        {
            float g0[kEP], g1[kEP];
#pragma unroll
            for (int q = 0; q < kEP; ++q) { g0[q] = t[0][q] * dsilu_f(a1[0][q]); g1[q] = t[1][q] * dsilu_f(a1[1][q]); }
            put(lane, g0); put(lane + 32, g1);
        }
        __syncwarp();
        float df[4] = { 0.f, 0.f, 0.f, 0.f };            // d f_k of edge el for k = kk + 4 c: sum over the 64 units in ascending order
#pragma unroll 8
        for (int i = 0; i < kH; ++i) {
            const float g = act[i * kEP + el];
            const float4 w = *reinterpret_cast<const float4 *>(W1Ts + i * kMaxRbf + kk * 4);
            df[0] = fmaf(g, w.x, df[0]); df[1] = fmaf(g, w.y, df[1]); df[2] = fmaf(g, w.z, df[2]); df[3] = fmaf(g, w.w, df[3]);
        }
        float dr = (df[0] * d[0] + df[1] * d[1]) + (df[2] * d[2] + df[3] * d[3]);
        dr += __shfl_xor_sync(0xffffffffu, dr, 1);
        dr += __shfl_xor_sync(0xffffffffu, dr, 2);
        if (kk == 0 && e0 + el < E) {
            const long long e = e0 + el;
            const float inv = r > 0.0f ? 1.0f / r : 0.0f;
            const float gx = dr * vx * inv, gy = dr * vy * inv, gz = dr * vz * inv;
            if (accumulate) { gvec[3 * e] += gx; gvec[3 * e + 1] += gy; gvec[3 * e + 2] += gz; }
            else { gvec[3 * e] = gx; gvec[3 * e + 1] = gy; gvec[3 * e + 2] = gz; }
        }
    }
}

constexpr int kHiddenSmemFwd = (kMaxRbf * kH + kH * kH + 4 * (kH * kEP + kMaxRbf * kEP)) * 4;
constexpr int kHiddenSmemBwd = (kMaxRbf * kH + 2 * kH * kH + kH * kMaxRbf + 4 * (kH * kEP + kMaxRbf * kEP)) * 4;

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

__device__ __forceinline__ float tf32_hi(float v) { return __uint_as_float(__float_as_uint(v) & 0xffffe000u); }

__device__ __forceinline__ void mbar_wait_parity(uint32_t bar, uint32_t parity)
{
    asm volatile("{\n.reg .pred p;\nLAB_WAIT:\nmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n@p bra DONE;\nbra LAB_WAIT;\nDONE:\n}"
                 :: "r"(bar), "r"(parity) : "memory");
}

// the three products of one K chunk (64 = 8 MMA steps of K = 8): lo*hi, hi*lo, hi*hi, smallest terms first
__device__ __forceinline__ void issue_chunk(uint32_t tmem_d, uint32_t sAhi, uint32_t sAlo, uint32_t sBhi, uint32_t sBlo, uint32_t idesc, bool first, int nprod = 3)
{
    if (nprod == 1) {           // measurement aid (E3_RADIAL_PRODUCTS=1): plain TF32, hi*hi only -- NOT fp32 accurate
#pragma unroll
        for (int ks = 0; ks < kTileK / 8; ++ks) {
            const uint64_t ahi = umma_desc(sAhi + ks * 256), bhi = umma_desc(sBhi + ks * 256);
            const uint32_t acc0 = (!first || ks > 0) ? 1u : 0u;
            asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n}"
                         :: "r"(tmem_d), "l"(ahi), "l"(bhi), "r"(idesc), "r"(acc0) : "memory");
        }
        return;
    }
#pragma unroll
    for (int ks = 0; ks < kTileK / 8; ++ks) {       // one MMA covers K = 8 (32 bytes = two core matrices): advance 256 bytes
        const uint64_t ahi = umma_desc(sAhi + ks * 256), alo = umma_desc(sAlo + ks * 256);
        const uint64_t bhi = umma_desc(sBhi + ks * 256), blo = umma_desc(sBlo + ks * 256);
        const uint32_t acc0 = (!first || ks > 0) ? 1u : 0u;
        asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n}"
                     :: "r"(tmem_d), "l"(alo), "l"(bhi), "r"(idesc), "r"(acc0) : "memory");
        asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n}"
                     :: "r"(tmem_d), "l"(ahi), "l"(blo), "r"(idesc), "r"(1u) : "memory");
        asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n}"
                     :: "r"(tmem_d), "l"(ahi), "l"(bhi), "r"(idesc), "r"(1u) : "memory");
    }
}

// TMEM -> registers -> shared-memory transpose -> global: warp w owns TMEM lanes 32 w .. 32 w + 31 (= tile rows).  A thread holds 32
// consecutive columns of ITS row; written out directly that is 16 bytes per lane at a row stride (half-filled sectors).  Each
// 32 x 32 block therefore goes through a per-warp staging buffer (row stride 36 floats: conflict-free both ways) and leaves as
// four full 128-byte row segments per store instruction.
template <int NT>
__device__ __forceinline__ void epilogue_tile(uint32_t tmem_d, int warp8, int lane, float *__restrict__ stg, float *__restrict__ D, long long ldd,
                                              long long m0, long long M, int n0, int N)
{
    // eight warps: warp8 % 4 selects the TMEM lane quarter (tile rows 32 q .. 32 q + 31), warp8 / 4 the column half
    const int warp = warp8 & 3;
    float *sw = stg + warp8 * (32 * 36);
#pragma unroll 1
    for (int c0 = (warp8 >> 2) * (NT / 2); c0 < (warp8 >> 2) * (NT / 2) + NT / 2; c0 += 32) {
        uint32_t v[32];
        const uint32_t taddr = tmem_d + ((uint32_t)(warp * 32) << 16) + (uint32_t)c0;
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 "
                     "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
                     "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
                     : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
                       "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]),
                       "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]),
                       "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
                     : "r"(taddr) : "memory");
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
        __syncwarp();
#pragma unroll
        for (int j = 0; j < 32; j += 4)
            *reinterpret_cast<float4 *>(sw + lane * 36 + j) = make_float4(__uint_as_float(v[j]), __uint_as_float(v[j + 1]), __uint_as_float(v[j + 2]), __uint_as_float(v[j + 3]));
        __syncwarp();
        const int col = n0 + c0 + 4 * (lane & 7);
#pragma unroll
        for (int it = 0; it < 8; ++it) {
            const int rl = it * 4 + (lane >> 3);
            const long long row = m0 + warp * 32 + rl;
            const float4 o = *reinterpret_cast<const float4 *>(sw + rl * 36 + 4 * (lane & 7));
            if (row < M) {
                float *dp = D + row * ldd + col;
                if (col + 4 <= N && (ldd & 3) == 0) __stcs(reinterpret_cast<float4 *>(dp), o);
                else {
                    if (col < N) dp[0] = o.x;
                    if (col + 1 < N) dp[1] = o.y;
                    if (col + 2 < N) dp[2] = o.z;
                    if (col + 3 < N) dp[3] = o.w;
                }
            }
        }
    }
}

// thread -> (row, 16-byte quad) of a [rows x 64] fp32 operand tile for pass j: a warp covers 8 consecutive rows x 4 consecutive quads,
// i.e. 64 contiguous bytes of 8 rows in global memory (whole sectors) and 512 contiguous bytes in the canonical shared-memory layout
// (conflict-free).  Eight warps: row = 16 j + 8 (warp / 4) + (lane & 7), quad = 4 (warp % 4) + (lane >> 3)
#define TILE_ROW(j) ((j) * 16 + (warp >> 2) * 8 + (lane & 7))
#define TILE_QUAD() ((warp & 3) * 4 + (lane >> 3))

// FORWARD, features as the M dimension:  D[f, e] = sum_k W3T[n_base + f, k] * h2[e, k]  for TWO slabs of 128 output features (A
// operands, staged once per CTA, 128 KB with their high / low parts) and a run of 64-edge tiles (B operand = the rows of h2, already
// split into TF32 high / low parts by the hidden kernel, brought in by 16-byte cp.async straight into the canonical layout).  Every B
// tile (32 KB through the L2 -> SM crossbar) now feeds 64 KB of output: the first version of this kernel kept one slab and a
// double-buffered B and was bound by exactly that traffic (91 GB of operand reads for 45.5 GB of output on config 4, every stall on
// an address register waiting for the LSU queue to drain, profiles/r02b).  In TMEM a lane is a FEATURE and a column an EDGE, so a
// tcgen05.ld leaves every warp with 32 consecutive features of one edge per register: each store instruction writes one full 128-byte
// line of w[e, n_base + ..] -- no shared-memory transpose.  Tiles are 64 edges so that B (2 x 32 KB) AND TMEM (2 x 128 columns) are
// double-buffered beside the 128 KB of slabs: the tensor core computes tile i while the eight warps drain tile i - 1 and the copies of
// tile i + 1 are in flight; one __syncthreads and one mbarrier wait per tile.
__global__ void __launch_bounds__(288, 1) radial_gemm_fwd_kernel(const float *__restrict__ Hhi, const float *__restrict__ Hlo, const float *__restrict__ W3Thi,
                                                                 const float *__restrict__ W3Tlo, float *__restrict__ D, long long ldd, long long E, int N,
                                                                 int tiles_per_cta, int nprod, int dbg)
{
    constexpr int NT = 64;                                                   // edges per tile (MMA N)
    extern __shared__ __align__(1024) unsigned char smem[];                  // [slab 0 hi | slab 0 lo | slab 1 hi | slab 1 lo] 32 KB each, then 3 x [B hi | B lo] 16 KB each
    __shared__ __align__(8) unsigned long long mbar[2];
    __shared__ uint32_t tmem_base_s;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int n_base = blockIdx.x * (2 * kTileM);
    const bool two = n_base + kTileM < N;                                    // the second slab holds features
    const long long n_etiles = (E + NT - 1) / NT;
    const long long t_begin = (long long)blockIdx.y * tiles_per_cta;
    const long long t_end = t_begin + tiles_per_cta < n_etiles ? t_begin + tiles_per_cta : n_etiles;
    if (t_begin >= t_end) return;
    const uint32_t mbar_s = (uint32_t)__cvta_generic_to_shared(&mbar[0]);
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 256;" :: "r"((uint32_t)__cvta_generic_to_shared(&tmem_base_s)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(mbar_s) : "memory");
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(mbar_s + 8) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    const uint32_t sA_s = (uint32_t)__cvta_generic_to_shared(smem), sB_s = sA_s + 131072;
    // warps 0-7 copy operands and drain TMEM; warp 8 only issues the MMAs (a ninth warp, so that no draining warp starts late)
    const bool worker = warp < 8;
    // stationary operands: 2 x 128 rows of W3^T (zero beyond N), high and low parts
    if (worker)
#pragma unroll
    for (int sl = 0; sl < 2; ++sl)
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const int row = TILE_ROW(j), q = TILE_QUAD();
            const uint32_t off = sl * 65536 + canon_off(row, q * 4);
            const int f = n_base + sl * kTileM + row;
            const bool v = f < N;
            const float *sh_ = W3Thi + (long long)(v ? f : 0) * kH + q * 4, *sl_ = W3Tlo + (long long)(v ? f : 0) * kH + q * 4;
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" :: "r"(sA_s + off), "l"(sh_), "r"(v ? 16 : 0) : "memory");
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" :: "r"(sA_s + 32768 + off), "l"(sl_), "r"(v ? 16 : 0) : "memory");
        }
    auto issue_b = [&](long long t, int buf) {
        if (!worker) return;
        if ((dbg & 4) || t >= t_end) { asm volatile("cp.async.commit_group;" ::: "memory"); return; }     // always one group per call
        const long long e0 = t * NT;
        const uint32_t bh = sB_s + buf * 32768, bl = bh + 16384;
#pragma unroll
        for (int j = 0; j < NT / 16; ++j) {
            const int row = TILE_ROW(j), q = TILE_QUAD();
            const uint32_t off = canon_off(row, q * 4);
            const bool v = e0 + row < E;
            const long long er = v ? e0 + row : 0;
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" :: "r"(bh + off), "l"(Hhi + er * kH + q * 4), "r"(v ? 16 : 0) : "memory");
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" :: "r"(bl + off), "l"(Hlo + er * kH + q * 4), "r"(v ? 16 : 0) : "memory");
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    issue_b(t_begin, 0);
    issue_b(t_begin + 1, 1);
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = tmem_base_s;
    const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(NT >> 3) << 17) | ((uint32_t)(kTileM >> 4) << 24);
    // warp -> (slab, TMEM lane quarter): it drains the 64 edge columns of its 32 features in two 32-column blocks
    const int slab = warp >> 2, quarter = warp & 3;
    const int feat = n_base + slab * kTileM + quarter * 32 + lane;           // this thread's output column of w
    auto epilogue = [&](long long t, int buf) {
        const long long e0 = t * NT;
        if (!worker || (slab == 1 && !two)) return;                          // warp-uniform
#pragma unroll 1
        for (int c0 = 0; c0 < NT; c0 += 32) {
            uint32_t v[32];
            const uint32_t taddr = tmem + buf * 128 + slab * 64 + ((uint32_t)(quarter * 32) << 16) + (uint32_t)c0;
            asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 "
                         "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
                         "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
                         : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
                           "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]),
                           "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]),
                           "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
                         : "r"(taddr) : "memory");
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
            if (feat < N && !(dbg & 1)) {
                float *dp = D + (e0 + c0) * ldd + feat;
                if (e0 + c0 + 32 <= E) {                 // whole block inside the graph: no per-store predicate
#pragma unroll
                    for (int j = 0; j < 32; ++j) { *dp = __uint_as_float(v[j]); dp += ldd; }
                } else {
#pragma unroll
                    for (int j = 0; j < 32; ++j)
                        if (e0 + c0 + j < E) dp[j * ldd] = __uint_as_float(v[j]);
                }
            }
        }
    };
    uint32_t ph0 = 0, ph1 = 0;
    // Tile t's B operand is copied two tiles ahead into a three-deep ring and its MMAs are issued right after the tile's barrier, i.e.
    // BEHIND the still running MMAs of tile t - 1: the tensor pipe never waits for a copy or a barrier.  The workers then wait for tile
    // t - 1 (its B buffer is the one tile t + 2 goes to, its accumulators are what they drain next).
    for (long long t = t_begin; t < t_end; ++t) {
        const int i = (int)(t - t_begin), bb = i % 3, tb = i & 1;
        asm volatile("cp.async.wait_group 1;" ::: "memory");                 // tile t (and, the first time, the slabs) has landed
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();                                                     // also: every warp has drained TMEM buffer `tb` (tile t - 2)
        if (tid == 256 && !(dbg & 2)) {
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            const uint32_t bh = sB_s + bb * 32768, bl = bh + 16384;
            issue_chunk(tmem + tb * 128, sA_s, sA_s + 32768, bh, bl, idesc, true, nprod);
            if (two) issue_chunk(tmem + tb * 128 + 64, sA_s + 65536, sA_s + 98304, bh, bl, idesc, true, nprod);
            asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(mbar_s + tb * 8) : "memory");
        }
        if (i > 0 && !(dbg & 2)) {                       // tile t - 1: MMAs done -> its B buffer is free, its accumulators are ready
            mbar_wait_parity(mbar_s + (tb ^ 1) * 8, (tb ^ 1) ? ph1 : ph0);
            if (tb ^ 1) ph1 ^= 1u; else ph0 ^= 1u;
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        }
        issue_b(t + 2, (i + 2) % 3);
        if (i > 0) epilogue(t - 1, tb ^ 1);
    }
    {
        const int tb = (int)((t_end - 1 - t_begin) & 1);
        if (!(dbg & 2)) mbar_wait_parity(mbar_s + tb * 8, tb ? ph1 : ph0);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        epilogue(t_end - 1, tb);
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 256;" :: "r"(tmem) : "memory");
}

// BACKWARD: D[128 NT-row tile, 64] = sum over K chunks of 64 / NT of A[rows x Kt] * B[64 x Kt]^T (A = grad_weights, fp32, streamed from
// HBM; B = W3 as TF32 high / low parts).  A CTA owns NT = 2 or 4 128-row MMA tiles (NT TMEM accumulators of 64 columns) that share every
// B chunk: each 256- or 512-row tile re-reads all of W3 (hi + lo, 1.1 MB on config 4) instead of each 128-row tile -- the first
// version's W3 traffic equalled its grad_weights traffic (45.5 GB each) and its time was set by the operand copies and the per-chunk
// synchronisation, not by the MMAs (radial GEMM experiments).  Chunks of K = 64 / NT keep the register staging (chunks
// kc + 1, kc + 2 in flight in registers while chunk kc is multiplied) and the shared-memory stages the size they were.  Canonical
// K-major no-swizzle layout with K-wide rows: core matrices of 8 rows x 16 bytes, 128 bytes apart along K (LBO), groups of 8 rows
// 32 K bytes apart (SBO).
template <int SBO>
__device__ __forceinline__ uint64_t umma_desc_sbo(uint32_t smem_addr)
{
    uint64_t d = 0;
    d |= (uint64_t)((smem_addr >> 4) & 0x3fff);
    d |= (uint64_t)((128u >> 4) & 0x3fff) << 16;
    d |= (uint64_t)(((uint32_t)SBO >> 4) & 0x3fff) << 32;
    d |= (uint64_t)1 << 46;
    return d;
}
template <int SBO>
__device__ __forceinline__ uint32_t canon_off_sbo(int row, int k)  // byte offset of element (row, k) of a [rows x SBO/32] fp32 tile
{
    return (uint32_t)((row >> 3) * SBO + (k >> 2) * 128 + (row & 7) * 16 + (k & 3) * 4);
}
// the three products of one K chunk (KS MMA steps of K = 8) of one 128-row tile: lo*hi, hi*lo, hi*hi
template <int KS, int SBO>
__device__ __forceinline__ void issue_chunk_t(uint32_t tmem_d, uint32_t sAhi, uint32_t sAlo, uint32_t sBhi, uint32_t sBlo, uint32_t idesc, bool first)
{
#pragma unroll
    for (int ks = 0; ks < KS; ++ks) {
        const uint64_t ahi = umma_desc_sbo<SBO>(sAhi + ks * 256), alo = umma_desc_sbo<SBO>(sAlo + ks * 256);
        const uint64_t bhi = umma_desc_sbo<SBO>(sBhi + ks * 256), blo = umma_desc_sbo<SBO>(sBlo + ks * 256);
        const uint32_t acc0 = (!first || ks > 0) ? 1u : 0u;
        asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n}"
                     :: "r"(tmem_d), "l"(alo), "l"(bhi), "r"(idesc), "r"(acc0) : "memory");
        asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n}"
                     :: "r"(tmem_d), "l"(ahi), "l"(blo), "r"(idesc), "r"(1u) : "memory");
        asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n}"
                     :: "r"(tmem_d), "l"(ahi), "l"(bhi), "r"(idesc), "r"(1u) : "memory");
    }
}

// NT 128-row MMA tiles per CTA and K chunks of KC (template parameters; rows x KC = 8192 elements per stage for <4,16> and <2,32>, one
// CTA per SM; <2,16,2> -- half the stage and register staging, TWO CTAs per SM -- was measured slower: 31.7 vs 27.4 ms on config 4)
template <int NT, int KC, int MINB>
__global__ void __launch_bounds__(256, MINB) radial_gemm_bwd_kernel(const float *__restrict__ A, long long lda, const float *__restrict__ Bhi,
                                                                 const float *__restrict__ Blo, long long ldb, float *__restrict__ D, long long M, long long Kt, int dbg)
{
    constexpr int kBwdTiles = NT;
    constexpr int kBwdRows = 128 * kBwdTiles, kBwdK = KC;
    constexpr int kBwdPA = NT * KC / 8;                                // 16-byte pieces of A per thread and chunk
    constexpr int kBwdPlane = kBwdRows * kBwdK * 4;                    // one A plane (high or low parts)
    constexpr int kBwdQPR = kBwdK / 4, kBwdPP = kBwdQPR / 4;           // 16-byte quads per row; passes per 64-row block
    constexpr int kBwdSBO = kBwdQPR * 128;                             // bytes between groups of 8 rows
    constexpr int kBwdB = 64 * kBwdK * 4;                              // one B plane
    constexpr int kBwdStage = 2 * kBwdPlane + 2 * kBwdB;               // stage: A hi | A lo | B hi | B lo
    extern __shared__ __align__(1024) unsigned char smem[];
    __shared__ __align__(8) unsigned long long mbar[2];
    __shared__ uint32_t tmem_base_s;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const long long m0 = (long long)blockIdx.x * kBwdRows;
    const uint32_t mbar_s = (uint32_t)__cvta_generic_to_shared(&mbar[0]);
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" :: "r"((uint32_t)__cvta_generic_to_shared(&tmem_base_s)), "n"(64 * kBwdTiles) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(mbar_s) : "memory");
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(mbar_s + 8) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = tmem_base_s;
    const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(kH >> 3) << 17) | ((uint32_t)(kTileM >> 4) << 24);
    const uint32_t smem_s = (uint32_t)__cvta_generic_to_shared(smem);
    const int k_chunks = (int)((Kt + kBwdK - 1) / kBwdK);
    // thread -> pieces of a chunk: A [256 x 8 quads]: pass j: row = (j / 2) * 64 + 8 warp + (lane & 7), quad = (j & 1) * 4 + (lane >> 3);
    // B [64 x 8 quads]: pass j: row = 8 warp + (lane & 7), quad = 4 j + (lane >> 3).  A warp covers 8 rows x 64 bytes: whole sectors in global
    // memory, 512 contiguous bytes in the canonical layout (conflict-free).
    const int r8 = warp * 8 + (lane & 7), q4 = lane >> 3;
    float4 ra0[kBwdPA], rbh0[kBwdPP], rbl0[kBwdPP], ra1[kBwdPA], rbh1[kBwdPP], rbl1[kBwdPP];
    auto load_chunk = [&](int kc, float4 (&ra)[kBwdPA], float4 (&rbh)[kBwdPP], float4 (&rbl)[kBwdPP]) {
        const long long k0 = (long long)kc * kBwdK;
#pragma unroll
        for (int j = 0; j < kBwdPA; ++j) {
            const int row = (j / kBwdPP) * 64 + r8, q = (j % kBwdPP) * 4 + q4;
            ra[j] = make_float4(0.f, 0.f, 0.f, 0.f);
            if (m0 + row < M && k0 + q * 4 + 4 <= Kt && !(dbg & 4)) ra[j] = __ldcs(reinterpret_cast<const float4 *>(A + (m0 + row) * lda + k0 + q * 4));
        }
#pragma unroll
        for (int j = 0; j < kBwdPP; ++j) {
            const int q = j * 4 + q4;
            rbh[j] = make_float4(0.f, 0.f, 0.f, 0.f); rbl[j] = rbh[j];
            if (k0 + q * 4 + 4 <= Kt && !(dbg & 8)) {
                rbh[j] = __ldg(reinterpret_cast<const float4 *>(Bhi + (long long)r8 * ldb + k0 + q * 4));
                rbl[j] = __ldg(reinterpret_cast<const float4 *>(Blo + (long long)r8 * ldb + k0 + q * 4));
            }
        }
    };
    auto store_chunk = [&](int buf, const float4 (&ra)[kBwdPA], const float4 (&rbh)[kBwdPP], const float4 (&rbl)[kBwdPP]) {
        unsigned char *base = smem + buf * kBwdStage;
#pragma unroll
        for (int j = 0; j < kBwdPA; ++j) {
            const int row = (j / kBwdPP) * 64 + r8, q = (j % kBwdPP) * 4 + q4;
            const float4 v = ra[j];
            const float4 h = make_float4(tf32_hi(v.x), tf32_hi(v.y), tf32_hi(v.z), tf32_hi(v.w));
            const uint32_t off = canon_off_sbo<kBwdSBO>(row, q * 4);
            *reinterpret_cast<float4 *>(base + off) = h;
            *reinterpret_cast<float4 *>(base + kBwdPlane + off) = make_float4(v.x - h.x, v.y - h.y, v.z - h.z, v.w - h.w);
        }
#pragma unroll
        for (int j = 0; j < kBwdPP; ++j) {
            const uint32_t off = canon_off_sbo<kBwdSBO>(r8, (j * 4 + q4) * 4);
            *reinterpret_cast<float4 *>(base + 2 * kBwdPlane + off) = rbh[j];
            *reinterpret_cast<float4 *>(base + 2 * kBwdPlane + kBwdB + off) = rbl[j];
        }
    };
    uint32_t ph0 = 0, ph1 = 0;
    auto step = [&](int kc, int buf, float4 (&ra)[kBwdPA], float4 (&rbh)[kBwdPP], float4 (&rbl)[kBwdPP], uint32_t &ph) {
        if (kc >= 2 && !(dbg & 1)) {                     // the MMAs of chunk kc - 2 must have finished reading this stage
            mbar_wait_parity(mbar_s + buf * 8, ph);
            ph ^= 1u;
        }
        if (!(dbg & 2)) store_chunk(buf, ra, rbh, rbl);
        if (kc + 2 < k_chunks) load_chunk(kc + 2, ra, rbh, rbl);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        if (tid == 0 && !(dbg & 1)) {
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            const uint32_t b = smem_s + buf * kBwdStage;
#pragma unroll
            for (int t = 0; t < kBwdTiles; ++t)          // tile t: rows 128 t .. 128 t + 127 of the stage, accumulator columns 64 t ..
                if (t == 0 || m0 + t * kTileM < M)
                    issue_chunk_t<kBwdK / 8, kBwdSBO>(tmem + 64 * t, b + t * 16 * kBwdSBO, b + kBwdPlane + t * 16 * kBwdSBO, b + 2 * kBwdPlane, b + 2 * kBwdPlane + kBwdB, idesc, kc == 0);
            asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(mbar_s + buf * 8) : "memory");
        }
    };
    load_chunk(0, ra0, rbh0, rbl0);
    if (k_chunks > 1) load_chunk(1, ra1, rbh1, rbl1);
    for (int kc = 0; kc < k_chunks; kc += 2) {
        step(kc, 0, ra0, rbh0, rbl0, ph0);
        if (kc + 1 < k_chunks) step(kc + 1, 1, ra1, rbh1, rbl1, ph1);
    }
    {   // the last commit covers every MMA issued before it
        const int buf = (k_chunks - 1) & 1;
        if (!(dbg & 1)) mbar_wait_parity(mbar_s + buf * 8, buf ? ph1 : ph0);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        float *stg = reinterpret_cast<float *>(smem + ((k_chunks & 1) ? kBwdStage : 0));       // the stage the last chunk did not use
        for (int t = 0; t < kBwdTiles; ++t)
            if (t == 0 || m0 + t * kTileM < M) epilogue_tile<kH>(tmem + 64 * t, warp, lane, stg, D, kH, m0 + t * kTileM, M, 0, kH);
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem), "n"(64 * kBwdTiles) : "memory");
}

// BACKWARD, warp-specialised version of the kernel above: NG groups of four producer warps and one MMA-issuing warp.  Group g owns
// shared-memory stage g and the K chunks kc = g (mod NG): it loads its chunk of grad_weights (and of W3) into registers, waits until
// the MMAs of its previous chunk have left the stage (empty[g], tcgen05.commit), splits and stores the chunk, fences the async proxy,
// arrives on full[g] (128 arrivals) and at once issues the loads of its next chunk; the MMA warp waits for full[g] chunk after chunk
// and issues the three products.  No block-wide barrier in the loop.
// What made the difference is the LANE MAPPING of the global loads (ncu on the lock-step kernel: L1 data-pipe LSU wavefronts at 96 %
// of peak, DRAM at 31 %): a 128-bit load is served a quarter-warp at a time, and with lanes 0-7 on eight different rows every quarter
// touched eight 128-byte lines -- 32 wavefronts per warp load.  Here consecutive lanes read consecutive 16-byte quads of ONE row
// (4 lanes x 64 bytes for KC = 16, 8 lanes x 128 bytes for KC = 32), so a quarter-warp touches two lines (one).  To keep the
// shared-memory stores of that mapping conflict-free the canonical layout is PADDED: core matrices (8 rows x 16 bytes) are LBO = 160
// (144) bytes apart along K instead of 128, so that the quads of a row fall into different 16-byte bank groups.
template <int LBO, int SBO>
__device__ __forceinline__ uint64_t umma_desc_pad(uint32_t smem_addr)
{
    uint64_t d = 0;
    d |= (uint64_t)((smem_addr >> 4) & 0x3fff);
    d |= (uint64_t)(((uint32_t)LBO >> 4) & 0x3fff) << 16;
    d |= (uint64_t)(((uint32_t)SBO >> 4) & 0x3fff) << 32;
    d |= (uint64_t)1 << 46;
    return d;
}
template <int KS, int LBO, int SBO>
__device__ __forceinline__ void issue_chunk_pad(uint32_t tmem_d, uint32_t sAhi, uint32_t sAlo, uint32_t sBhi, uint32_t sBlo, uint32_t idesc, bool first)
{
#pragma unroll
    for (int ks = 0; ks < KS; ++ks) {
        const uint64_t ahi = umma_desc_pad<LBO, SBO>(sAhi + ks * 2 * LBO), alo = umma_desc_pad<LBO, SBO>(sAlo + ks * 2 * LBO);
        const uint64_t bhi = umma_desc_pad<LBO, SBO>(sBhi + ks * 2 * LBO), blo = umma_desc_pad<LBO, SBO>(sBlo + ks * 2 * LBO);
        const uint32_t acc0 = (!first || ks > 0) ? 1u : 0u;
        asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n}"
                     :: "r"(tmem_d), "l"(alo), "l"(bhi), "r"(idesc), "r"(acc0) : "memory");
        asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n}"
                     :: "r"(tmem_d), "l"(ahi), "l"(blo), "r"(idesc), "r"(1u) : "memory");
        asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n}"
                     :: "r"(tmem_d), "l"(ahi), "l"(bhi), "r"(idesc), "r"(1u) : "memory");
    }
}

template <int NT, int KC, int NG>
__global__ void __launch_bounds__(128 * NG + 32, 1) radial_gemm_bwd_pp_kernel(const float *__restrict__ A, long long lda, const float *__restrict__ Bhi,
                                                                            const float *__restrict__ Blo, long long ldb, float *__restrict__ D, long long M, long long Kt, int dbg)
{
    constexpr int kRows = 128 * NT;
    constexpr int kQPR = KC / 4;                                       // 16-byte quads per row of a chunk = lanes per row (4 or 8)
    static_assert(kQPR == 4 || kQPR == 8, "KC must be 16 or 32");
    constexpr int kLBO = kQPR == 4 ? 160 : 144;                        // padded K stride of the core matrices (see above)
    constexpr int kSBO = kQPR * kLBO;                                  // bytes between groups of 8 rows
    constexpr int kPlane = (kRows / 8) * kSBO, kB = 8 * kSBO;
    constexpr int kStage = 2 * kPlane + 2 * kB;                        // A hi | A lo | B hi | B lo
    constexpr int kRPI = 32 / kQPR;                                    // rows per warp instruction (8 or 4)
    constexpr int kRPP = 4 * kRPI;                                     // rows per pass of a four-warp group (32 or 16)
    constexpr int kPA = kRows / kRPP, kPB = 64 / kRPP;                 // 16-byte pieces of A / of each B plane per producer thread and chunk
    extern __shared__ __align__(1024) unsigned char smem[];
    __shared__ __align__(8) unsigned long long mbar[2 * NG + 1];       // full[NG], empty[NG], done
    __shared__ uint32_t tmem_base_s;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const long long m0 = (long long)blockIdx.x * kRows;
    const uint32_t mbar_s = (uint32_t)__cvta_generic_to_shared(&mbar[0]);
    const uint32_t full_s = mbar_s, empty_s = mbar_s + 8 * NG, done_s = mbar_s + 16 * NG;
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" :: "r"((uint32_t)__cvta_generic_to_shared(&tmem_base_s)), "n"(64 * NT) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    if (tid == 0) {
        for (int g = 0; g < NG; ++g) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 128;" :: "r"(full_s + 8 * g) : "memory");
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(empty_s + 8 * g) : "memory");
        }
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(done_s) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = tmem_base_s;
    const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(kH >> 3) << 17) | ((uint32_t)(kTileM >> 4) << 24);
    const uint32_t smem_s = (uint32_t)__cvta_generic_to_shared(smem);
    const int k_chunks = (int)((Kt + KC - 1) / KC);
    if (warp == 4 * NG) {
        if (lane == 0) {
            for (int kc = 0; kc < k_chunks; ++kc) {
                const int g = kc % NG;
                mbar_wait_parity(full_s + 8 * g, (uint32_t)((kc / NG) & 1));
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const uint32_t b = smem_s + g * kStage;
#pragma unroll
                for (int t = 0; t < NT; ++t)
                    if ((t == 0 || m0 + t * kTileM < M) && !(dbg & 8))
                        issue_chunk_pad<KC / 8, kLBO, kSBO>(tmem + 64 * t, b + t * 16 * kSBO, b + kPlane + t * 16 * kSBO, b + 2 * kPlane, b + 2 * kPlane + kB, idesc, kc == 0);
                asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(empty_s + 8 * g) : "memory");
            }
            asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(done_s) : "memory");
        }
    } else {
        const int g = warp >> 2;
        const int rl = (warp & 3) * kRPI + lane / kQPR, ql = lane % kQPR;          // row within a pass, quad within the row
        const uint32_t off0 = (uint32_t)((rl >> 3) * kSBO + ql * kLBO + (rl & 7) * 16);
        constexpr uint32_t kOffPass = (uint32_t)((kRPP / 8) * kSBO);               // kRPP is a multiple of 8: whole row groups per pass
        float4 ra[kPA], rbh[kPB], rbl[kPB];
        auto load_chunk = [&](int kc) {
            const long long k0 = (long long)kc * KC + ql * 4;
            const bool kok = k0 + 4 <= Kt;
#pragma unroll
            for (int j = 0; j < kPA; ++j) {
                const long long row = m0 + j * kRPP + rl;
                ra[j] = make_float4(0.f, 0.f, 0.f, 0.f);
                if (row < M && kok && !(dbg & 2)) ra[j] = __ldcs(reinterpret_cast<const float4 *>(A + row * lda + k0));
            }
#pragma unroll
            for (int j = 0; j < kPB; ++j) {
                const int row = j * kRPP + rl;
                rbh[j] = make_float4(0.f, 0.f, 0.f, 0.f); rbl[j] = rbh[j];
                if (kok) {
                    rbh[j] = __ldg(reinterpret_cast<const float4 *>(Bhi + (long long)row * ldb + k0));
                    rbl[j] = __ldg(reinterpret_cast<const float4 *>(Blo + (long long)row * ldb + k0));
                }
            }
        };
        unsigned char *base = smem + g * kStage;
        uint32_t ph = 0;
        if (g < k_chunks) load_chunk(g);
        for (int kc = g; kc < k_chunks; kc += NG) {
            if (kc >= NG) {                              // the MMAs of this group's previous chunk must have finished reading the stage
                mbar_wait_parity(empty_s + 8 * g, ph);
                ph ^= 1u;
            }
            if (!(dbg & 4)) {
#pragma unroll
                for (int j = 0; j < kPA; ++j) {
                    const float4 v = ra[j];
                    const float4 h = make_float4(tf32_hi(v.x), tf32_hi(v.y), tf32_hi(v.z), tf32_hi(v.w));
                    const uint32_t off = off0 + j * kOffPass;
                    *reinterpret_cast<float4 *>(base + off) = h;
                    *reinterpret_cast<float4 *>(base + kPlane + off) = make_float4(v.x - h.x, v.y - h.y, v.z - h.z, v.w - h.w);
                }
            }
#pragma unroll
            for (int j = 0; j < kPB; ++j) {
                const uint32_t off = off0 + j * kOffPass;
                *reinterpret_cast<float4 *>(base + 2 * kPlane + off) = rbh[j];
                *reinterpret_cast<float4 *>(base + 2 * kPlane + kB + off) = rbl[j];
            }
            if (!(dbg & 1)) asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(full_s + 8 * g) : "memory");
            if (kc + NG < k_chunks) load_chunk(kc + NG);
        }
        mbar_wait_parity(done_s, 0u);                   // every MMA has finished: accumulators complete, all stages free
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        if (warp < 8) {
            float *stg = reinterpret_cast<float *>(smem);
            for (int t = 0; t < NT; ++t)
                if (t == 0 || m0 + t * kTileM < M) epilogue_tile<kH>(tmem + 64 * t, warp, lane, stg, D, kH, m0 + t * kTileM, M, 0, kH);
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem), "n"(64 * NT) : "memory");
}

constexpr int kGemmSmemFwd = 229376;   // forward: 2 x 64 KB of A + 3 x 32 KB of B
constexpr int kGemmSmem = 196608;      //; backward: 2 x 96 KB stages (the epilogue stages through an idle buffer)

int launch_gemm_fwd(const float *Hhi, const float *Hlo, const float *W3Thi, const float *W3Tlo, float *D, long long ldd, long long E, int N, cudaStream_t st)
{
    static bool attr_set = false;
    if (!attr_set) {
        E3_CUDA_TRY(cudaFuncSetAttribute(radial_gemm_fwd_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kGemmSmemFwd));
        E3_CUDA_TRY(cudaFuncSetAttribute(radial_gemm_bwd_kernel<4, 16, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, kGemmSmem));
        E3_CUDA_TRY(cudaFuncSetAttribute(radial_gemm_bwd_kernel<2, 32, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, kGemmSmem));
        attr_set = true;
    }
    if (E <= 0) return E3_OK;
    // grid: (pairs of 128-feature slabs) x (runs of edge tiles): a CTA keeps its slabs for `tiles_per_cta` 64-edge tiles; enough CTAs for
    // ~8 per SM so that the slabs of one edge range run together (the h2 rows they share stay in L2)
    const int slabs = (N + 2 * kTileM - 1) / (2 * kTileM);       // pairs of 128-feature slabs
    const long long n_etiles = (E + 63) / 64;
    long long runs = (148LL * 8 + slabs - 1) / slabs;
    if (runs > n_etiles) runs = n_etiles;
    const int tiles_per_cta = (int)((n_etiles + runs - 1) / runs);
    runs = (n_etiles + tiles_per_cta - 1) / tiles_per_cta;
    if (runs > 65535) { set_error("radial gemm: grid too large"); return E3_ERR_UNSUPPORTED; }
    static const int nprod = []() { const char *e = getenv("E3_RADIAL_PRODUCTS"); return (e && e[0] == '1') ? 1 : 3; }();
    static const int dbg = []() { const char *e = getenv("E3_RADIAL_DBG"); return e ? atoi(e) : 0; }();
    radial_gemm_fwd_kernel<<<dim3((unsigned)slabs, (unsigned)runs), 288, kGemmSmemFwd, st>>>(Hhi, Hlo, W3Thi, W3Tlo, D, ldd, E, N, tiles_per_cta, nprod, dbg);
    E3_CUDA_TRY(cudaGetLastError());
    return E3_OK;
}

int launch_gemm_bwd(const float *A, long long lda, const float *Bhi, const float *Blo, long long ldb, float *D, long long M, long long Kt, cudaStream_t st)
{
    static bool attr_set = false;
    if (!attr_set) {
        E3_CUDA_TRY(cudaFuncSetAttribute(radial_gemm_fwd_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kGemmSmemFwd));
        E3_CUDA_TRY(cudaFuncSetAttribute(radial_gemm_bwd_kernel<4, 16, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, kGemmSmem));
        E3_CUDA_TRY(cudaFuncSetAttribute(radial_gemm_bwd_kernel<2, 32, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, kGemmSmem));
        attr_set = true;
    }
    if (M <= 0) return E3_OK;
    // 512-row CTAs once they still give the machine four waves (every CTA re-reads all of W3), 256-row CTAs below that
    const int nt = M >= 4LL * 148 * 512 ? 4 : 2;
    const long long grid = (M + 128 * nt - 1) / (128 * nt);
    if (grid > 0x7fffffffLL) { set_error("radial gemm: grid too large"); return E3_ERR_UNSUPPORTED; }
    static const int dbg = []() { const char *e = getenv("E3_RADIAL_DBG_BWD"); return e ? atoi(e) : 0; }();
    static const int pp = []() { const char *e = getenv("E3_RADIAL_BWD_PP"); return e ? atoi(e) : 1; }();      // 0 = the lock-step kernel above
    if (pp) {
        constexpr int kPPSmem = 2 * 92160;       // two padded stages (either shape)
        static bool pp_attr = false;
        if (!pp_attr) {
            E3_CUDA_TRY(cudaFuncSetAttribute(radial_gemm_bwd_pp_kernel<4, 16, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, kPPSmem));
            E3_CUDA_TRY(cudaFuncSetAttribute(radial_gemm_bwd_pp_kernel<2, 32, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, kPPSmem));
            pp_attr = true;
        }
        // 256 rows x K chunks of 32 (a row's 128-byte line per chunk) everywhere: config 4 18.2 ms against 19.4 for 512 x 16, config 2 0.284
        // against 0.363 (whole radial backward); E3_RADIAL_BWD_PP=16 selects the 512 x 16 shape, =0 the lock-step kernel (measurement aids)
        const bool wide = pp != 16;
        const long long grid2 = wide ? (M + 255) / 256 : (M + 511) / 512;
        if (!wide) radial_gemm_bwd_pp_kernel<4, 16, 2><<<(unsigned)grid2, 288, kPPSmem, st>>>(A, lda, Bhi, Blo, ldb, D, M, Kt, dbg);
        else radial_gemm_bwd_pp_kernel<2, 32, 2><<<(unsigned)grid2, 288, kPPSmem, st>>>(A, lda, Bhi, Blo, ldb, D, M, Kt, dbg);
        E3_CUDA_TRY(cudaGetLastError());
        return E3_OK;
    }
    if (nt == 4) radial_gemm_bwd_kernel<4, 16, 1><<<(unsigned)grid, 256, kGemmSmem, st>>>(A, lda, Bhi, Blo, ldb, D, M, Kt, dbg);
    else radial_gemm_bwd_kernel<2, 32, 1><<<(unsigned)grid, 256, kGemmSmem, st>>>(A, lda, Bhi, Blo, ldb, D, M, Kt, dbg);
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
    return (size_t)n_edges * kH * sizeof(float) * 2 + 256;   // h2 as TF32 high / low parts (forward), dh2 (backward): [E,64] fp32 each
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
    const long long blocks = std::min<long long>((n_edges + 31) / 32, 148LL * 8);
    radial_hidden_kernel<false><<<(unsigned)blocks, 128, kHiddenSmemFwd, st>>>(vec, n_edges, net->K, net->p, (float)net->rc, net->W1, net->W2, net->W2T, h2,
                                                                                nullptr, nullptr, 0);
    E3_CUDA_TRY(cudaGetLastError());
    return launch_gemm_fwd(h2, h2 + (size_t)n_edges * kH, net->W3T_hi, net->W3T_lo, weights, net->n_out, n_edges, net->n_out, st);
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
    int rc = launch_gemm_bwd(grad_weights, net->n_out, net->W3_hi, net->W3_lo, net->n_out, dh2, n_edges, net->n_out, st);
    if (rc != E3_OK) return rc;
    const long long blocks = std::min<long long>((n_edges + 31) / 32, 148LL * 8);
    static bool hidden_attr = false;
    if (!hidden_attr) {          // 50 KB of dynamic shared memory: above the 48 KB default
        E3_CUDA_TRY(cudaFuncSetAttribute(radial_hidden_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kHiddenSmemBwd));
        hidden_attr = true;
    }
    radial_hidden_kernel<true><<<(unsigned)blocks, 128, kHiddenSmemBwd, st>>>(vec, n_edges, net->K, net->p, (float)net->rc, net->W1, net->W2, net->W2T, nullptr,
                                                                               dh2, grad_vec, accumulate);
    E3_CUDA_TRY(cudaGetLastError());
    return E3_OK;
}
