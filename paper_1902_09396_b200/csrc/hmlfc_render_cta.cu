// Fused decode + render kernel with the tile tables built inside the CTA and a quadtree of sub-tile passes (sm_100a): renders every
// tile hmlfc_render_tiles.cu hands over and whole views at low magnification (about as many light-field samples as output pixels
// under a tile, or more).  For B = 4 streams.
//
// PAPER.md:289-293 (decoding procedure), :309 (random access), :73 / :409 (two-plane rendering); definitions: DESIGN.md sections 3
// and 5; phases and vocabulary: hmlfc_render_common.cuh.
//
// One CTA of NT threads renders a TW x TH tile of one output view, 4 consecutive pixels per thread (NT = 256: 32 x 32,
// NT = 512: 64 x 32, NT = 1024: 64 x 64):
//   A   ray set-up (screen coordinates once per column / row, shared by shuffles), 16-tap footprint per pixel;
//   SV  integer (u,v) range and (s,t) box of the tile's taps (warp reductions + 8 shared atomics per warp);
//   T   warp 0 builds the view table, warp 1 the plane table, the other warps zero the accumulators;
//   B1 - B4, C  as in hmlfc_render_common.cuh.
// A tile whose tables do not fit the shared-memory arena (minification) is rendered as its four quadrants with one pixel
// per thread, a quadrant that does not fit is split again, down to 8-pixel-wide sub-tiles; one of those that still does
// not fit is rendered by 16 direct sample decodes per pixel.  All paths produce identical bytes.
#include "hmlfc_render_common.cuh"

namespace hmlfc {

namespace {

template <int kArenaBytes, int kMinBlocks, int kNT, int kTW>
__global__ void __launch_bounds__(kNT, kMinBlocks)
render_cta_kernel(const __grid_constant__ DevStream S, const Camera *__restrict__ cams, int W, int H, uint8_t *__restrict__ out, int out_aligned)
{
    extern __shared__ __align__(16) unsigned char arena[];
    __shared__ Ctl ctl;
    const int tid = threadIdx.x;
    const int view = blockIdx.z;
    for (int q = tid; q < 192; q += kNT)
        reinterpret_cast<uint32_t *>(ctl.lut)[q] = reinterpret_cast<const uint32_t *>(g_cta_digit_lut.v)[q];
    reset_ctl(ctl);
    // the camera goes to shared memory (16 registers per thread otherwise, or reloads from global memory in every pass)
    if (tid < 16) reinterpret_cast<float *>(&ctl.cam)[tid] = reinterpret_cast<const float *>(cams + view)[tid];
    __syncthreads();
    if (tid < 2) camera_affine(S, ctl.cam, tid, ctl.aff[tid]);
    render_tile_general<kArenaBytes, kNT, kTW>(S, ctl, arena, W, H, out, out_aligned, view, (int)blockIdx.x, (int)blockIdx.y);
}

}  // namespace

#ifdef HMLFC_PASS_STATS
extern "C" int hmlfc_debug_pass_stats(unsigned long long *out, int reset)
{
    cudaDeviceSynchronize();
    cudaMemcpyFromSymbol(out, g_pass_stats, sizeof(g_pass_stats));
    if (reset) { unsigned long long z[64] = {}; cudaMemcpyToSymbol(g_pass_stats, z, sizeof(z)); }
    return 0;
}
#endif

// Shared memory per SM: 233,472 bytes, 1 KB reserved per resident CTA, 9.4 KB of tables (Ctl) per CTA; the rest is the arena.
//   0: 256 threads, 32 x 32 tile, 3 CTAs x 65 KB     1: 256 threads, 32 x 32 tile, 2 CTAs x 103 KB (views that look at about as many
//   2: 256 threads, 32 x 32 tile, 4 CTAs x 46 KB        light-field samples as they have pixels: far fewer tiles are split)
//   3: 1024 threads, 64 x 64 tile, 1 CTA x 200 KB    4: 512 threads, 64 x 32 tile, 2 CTAs x 100 KB
#ifndef HMLFC_ARENA3_KB
#define HMLFC_ARENA3_KB 200
#endif
#ifndef HMLFC_ARENA4_KB
#define HMLFC_ARENA4_KB 100
#endif
#define HMLFC_CTA_CONFIGS(X) \
    X(0, 65 * 1024, 3, 256, 32) \
    X(1, 103 * 1024, 2, 256, 32) \
    X(2, 46 * 1024, 4, 256, 32) \
    X(3, HMLFC_ARENA3_KB * 1024, 1, 1024, 64) \
    X(4, HMLFC_ARENA4_KB * 1024, 2, 512, 64)

cudaError_t configure_render_cta()
{
    cudaError_t e = cudaSuccess;
#define X(id, arena, minb, nt, tw) \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(render_cta_kernel<arena, minb, nt, tw>, cudaFuncAttributeMaxDynamicSharedMemorySize, arena);
    HMLFC_CTA_CONFIGS(X)
#undef X
    return e;
}

cudaError_t launch_render_cta(const DevStream &S, const Camera *d_cams, int n_views, int W, int H, uint8_t *d_out, cudaStream_t st,
                              int *n_launches, int config)
{
    if (n_views == 0) return cudaSuccess;
    if (S.B != 4) return cudaErrorInvalidValue;  // block-row tasks are written for 4 x 4 blocks; the caller dispatches other sizes elsewhere
    const int aligned = ((reinterpret_cast<uintptr_t>(d_out) & 3u) == 0 && (W % 4) == 0) ? 1 : 0;
    if (config < 0) config = (long long)W * H < 2LL * S.Ws * S.Ht ? 1 : ((long long)W * H >= 8LL * S.Ws * S.Ht ? 2 : 0);
    cudaError_t e = cudaErrorInvalidValue;
#define X(id, arena, minb, nt, tw) \
    if (config == id) { \
        constexpr int th = nt * kPPL / tw; \
        dim3 grid((unsigned)((W + tw - 1) / tw), (unsigned)((H + th - 1) / th), (unsigned)n_views); \
        if (grid.y > 65535u) return cudaErrorInvalidValue; \
        render_cta_kernel<arena, minb, nt, tw><<<grid, dim3(nt), arena, st>>>(S, d_cams, W, H, d_out, aligned); \
        e = cudaGetLastError(); \
    }
    HMLFC_CTA_CONFIGS(X)
#undef X
    if (n_launches && e == cudaSuccess) *n_launches += 1;
    return e;
}

}  // namespace hmlfc
