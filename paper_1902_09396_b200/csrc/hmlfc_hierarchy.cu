// hmlfc_hierarchy: forward colour transform + RLFC hierarchy build of the HMLFC encoder on sm_100a (SURVEY.md 8(f) rank 1,
// "hierarchy build"; the companion of hmlfc_search).
//
// the views are converted to YCoCg ("to avoid any loss of information": the reversible lifting form,
// DESIGN.md R17); PAPER.md:200 (section 4.3): the views are clustered by their position on the camera grid (2 x 2, R1), the
// representative key view (RKV) of a cluster is the pixel-wise filtered cluster (uniform mean of the members present, rounded
// half away from zero, R2 / R3) and each member's sparse residual view is SRV = member - RKV; the RKVs are clustered again
// up to the tree height.  Identity: X_0[p] = X_h[p >> h] + sum_L SRV_L[p >> L].
//
// Pure streaming work, bound by HBM: every kernel reads each input sample once and writes each output sample once, four
// consecutive pixels per thread (12-byte RGB reads, 8-byte int16x4 reads and writes), a warp's accesses contiguous per
// stream.  Level 0 is fused with the colour transform (X_0 is never written: only SRV_0 and X_1 leave the kernel).
// Algorithmic bytes per light-field pixel: 3 read + 6 (SRV_0) + 1.5 (X_1) written, then per level L >= 1 and plane pixel
// 6 read + 6 + 1.5 written on 4^-L of the pixels.  Integer arithmetic, bit-exact against the oracle's encoder.
#include <cuda_runtime.h>
#include <stdint.h>

#include "hmlfc.h"

namespace hmlfc {

namespace {

constexpr int kThreads = 256;

// round(sum / n), half away from zero, n in {1, 2, 4}
__device__ __forceinline__ int round_mean(int sum, int n)
{
    const int a = sum < 0 ? -sum : sum;
    const int q = n == 4 ? (a + 2) >> 2 : (n == 2 ? (a + 1) >> 1 : a);
    return sum < 0 ? -q : q;
}

__device__ __forceinline__ uint2 pack4(const int v[4])
{
    return make_uint2(((uint32_t)v[0] & 0xFFFFu) | ((uint32_t)v[1] << 16), ((uint32_t)v[2] & 0xFFFFu) | ((uint32_t)v[3] << 16));
}

__device__ __forceinline__ void unpack4(uint2 w, int v[4])
{
    v[0] = (int)(int16_t)(w.x & 0xFFFFu); v[1] = (int)w.x >> 16;
    v[2] = (int)(int16_t)(w.y & 0xFFFFu); v[3] = (int)w.y >> 16;
}

// level 0: RGB8 views -> SRV_0 of every view and X_1 of every cluster, 4 consecutive pixels of one cluster per thread.
// npx4 = Ws * Ht / 4.  Plane strides are in samples (npx = Ws * Ht).
#ifndef HMLFC_HIER_MINB
#define HMLFC_HIER_MINB 4
#endif
__global__ void __launch_bounds__(kThreads, HMLFC_HIER_MINB)
level0_kernel(const uint8_t *__restrict__ lf, int U, int V, int U1, size_t npx, size_t srv_ch_stride, size_t x_ch_stride,
              int16_t *__restrict__ srv0, int16_t *__restrict__ x1)
{
    const size_t i4 = (size_t)blockIdx.x * kThreads + threadIdx.x;
    if (i4 * 4 >= npx) return;
    const int q = blockIdx.y, qv = q / U1, qu = q - qv * U1;
    int val[4][3][4];  // member, channel, pixel
    int sum[3][4] = {};
    int n = 0;
    bool present[4];
#pragma unroll
    for (int mbr = 0; mbr < 4; ++mbr) {
        const int pu = 2 * qu + (mbr & 1), pv = 2 * qv + (mbr >> 1);
        present[mbr] = pu < U && pv < V;
        if (!present[mbr]) continue;
        ++n;
        const uint32_t *p = reinterpret_cast<const uint32_t *>(lf + ((size_t)(pv * U + pu) * npx + i4 * 4) * 3);
        const uint32_t w0 = __ldg(p), w1 = __ldg(p + 1), w2 = __ldg(p + 2);  // 4 RGB triples = 12 bytes
        const int r[4] = {(int)(w0 & 0xFF), (int)(w0 >> 24), (int)((w1 >> 16) & 0xFF), (int)((w2 >> 8) & 0xFF)};
        const int g[4] = {(int)((w0 >> 8) & 0xFF), (int)(w1 & 0xFF), (int)(w1 >> 24), (int)((w2 >> 16) & 0xFF)};
        const int b[4] = {(int)((w0 >> 16) & 0xFF), (int)((w1 >> 8) & 0xFF), (int)(w2 & 0xFF), (int)(w2 >> 24)};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            // forward YCoCg-R (arithmetic shifts = floor)
            const int co = r[k] - b[k];
            const int t = b[k] + (co >> 1);
            const int cg = g[k] - t;
            const int y = t + (cg >> 1);
            val[mbr][0][k] = y; val[mbr][1][k] = co; val[mbr][2][k] = cg;
            sum[0][k] += y; sum[1][k] += co; sum[2][k] += cg;
        }
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        int rk[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) rk[k] = round_mean(sum[c][k], n);  // RKV = filtered cluster
        *reinterpret_cast<uint2 *>(x1 + (size_t)c * x_ch_stride + (size_t)q * npx + i4 * 4) = pack4(rk);
#pragma unroll
        for (int mbr = 0; mbr < 4; ++mbr) {
            if (!present[mbr]) continue;
            const int pu = 2 * qu + (mbr & 1), pv = 2 * qv + (mbr >> 1);
            int d[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) d[k] = val[mbr][c][k] - rk[k];  // SRV = member - RKV
            *reinterpret_cast<uint2 *>(srv0 + (size_t)c * srv_ch_stride + (size_t)(pv * U + pu) * npx + i4 * 4) = pack4(d);
        }
    }
}

// level L >= 1: X_L planes -> SRV_L of every plane and X_{L+1} of every cluster; blockIdx.z = channel
__global__ void __launch_bounds__(kThreads)
levelL_kernel(const int16_t *__restrict__ xl, int UL, int VL, int UN, size_t npx, size_t x_ch_stride, size_t srv_ch_stride,
              int16_t *__restrict__ srvl, int16_t *__restrict__ xn)
{
    const size_t i4 = (size_t)blockIdx.x * kThreads + threadIdx.x;
    if (i4 * 4 >= npx) return;
    const int q = blockIdx.y, qv = q / UN, qu = q - qv * UN, c = blockIdx.z;
    const int16_t *xc = xl + (size_t)c * x_ch_stride;
    int val[4][4], sum[4] = {0, 0, 0, 0}, n = 0;
    bool present[4];
#pragma unroll
    for (int mbr = 0; mbr < 4; ++mbr) {
        const int pu = 2 * qu + (mbr & 1), pv = 2 * qv + (mbr >> 1);
        present[mbr] = pu < UL && pv < VL;
        if (!present[mbr]) continue;
        ++n;
        unpack4(__ldg(reinterpret_cast<const uint2 *>(xc + (size_t)(pv * UL + pu) * npx + i4 * 4)), val[mbr]);
#pragma unroll
        for (int k = 0; k < 4; ++k) sum[k] += val[mbr][k];
    }
    int rk[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) rk[k] = round_mean(sum[k], n);
    *reinterpret_cast<uint2 *>(xn + (size_t)c * x_ch_stride + (size_t)q * npx + i4 * 4) = pack4(rk);
#pragma unroll
    for (int mbr = 0; mbr < 4; ++mbr) {
        if (!present[mbr]) continue;
        const int pu = 2 * qu + (mbr & 1), pv = 2 * qv + (mbr >> 1);
        int d[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) d[k] = val[mbr][k] - rk[k];
        *reinterpret_cast<uint2 *>(srvl + (size_t)c * srv_ch_stride + (size_t)(pv * UL + pu) * npx + i4 * 4) = pack4(d);
    }
}

}  // namespace

}  // namespace hmlfc

extern "C" int hmlfc_hierarchy_sizes(int U, int V, int height, int64_t *n_srv_planes, int64_t *n_x_planes)
{
    if (U < 1 || V < 1 || height < 1 || height > 8 || !n_srv_planes || !n_x_planes) return HMLFC_E_INVALID;
    int64_t ns = 0, nx = 0;
    for (int L = 0; L <= height; ++L) {
        const int64_t n = (int64_t)((U + (1 << L) - 1) >> L) * ((V + (1 << L) - 1) >> L);
        if (L < height) ns += n;
        if (L >= 1) nx += n;
    }
    *n_srv_planes = ns;
    *n_x_planes = nx;
    return HMLFC_OK;
}

extern "C" int hmlfc_hierarchy(const uint8_t *d_lf, int U, int V, int Ws, int Ht, int height, int16_t *d_srv, int16_t *d_x,
                               void *cuda_stream)
{
    using namespace hmlfc;
    int64_t ns = 0, nx = 0;
    if (!d_lf || !d_srv || !d_x || Ws < 1 || Ht < 1 || hmlfc_hierarchy_sizes(U, V, height, &ns, &nx) != HMLFC_OK) return HMLFC_E_INVALID;
    if (Ws % 4) return HMLFC_E_UNSUPPORTED;  // four pixels per thread (every configuration has B = 4 | Ws)
    if ((reinterpret_cast<uintptr_t>(d_lf) & 3u) || (reinterpret_cast<uintptr_t>(d_srv) & 7u) || (reinterpret_cast<uintptr_t>(d_x) & 7u))
        return HMLFC_E_INVALID;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const size_t npx = (size_t)Ws * Ht;
    const size_t srv_ch = (size_t)ns * npx, x_ch = (size_t)nx * npx;
    const unsigned gx = (unsigned)((npx / 4 + kThreads - 1) / kThreads);
    int UL = U, VL = V;
    size_t srv_off = 0, x_off = 0;  // plane offsets of the level being written (SRV_L) / read (X_L, L >= 1)
    for (int L = 0; L < height; ++L) {
        const int UN = (UL + 1) >> 1, VN = (VL + 1) >> 1;
        if ((long long)UN * VN > 65535) return HMLFC_E_UNSUPPORTED;
        if (L == 0) {
            level0_kernel<<<dim3(gx, (unsigned)(UN * VN)), kThreads, 0, st>>>(d_lf, U, V, UN, npx, srv_ch, x_ch, d_srv, d_x);
        } else {
            const size_t xn_off = x_off + (size_t)UL * VL;
            levelL_kernel<<<dim3(gx, (unsigned)(UN * VN), 3), kThreads, 0, st>>>(d_x + x_off * npx, UL, VL, UN, npx, x_ch, srv_ch,
                                                                                 d_srv + srv_off * npx, d_x + xn_off * npx);
            x_off = xn_off;
        }
        srv_off += (size_t)UL * VL;
        UL = UN; VL = VN;
    }
    return cudaGetLastError() == cudaSuccess ? HMLFC_OK : HMLFC_E_CUDA;
}
