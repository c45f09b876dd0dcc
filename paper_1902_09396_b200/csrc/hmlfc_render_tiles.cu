// Fused decode + render for B = 4 streams, default path of hmlfc_render (sm_100a): tile tables from a kernel of their own, one pass
// per 32 x 32 tile.
//
// PAPER.md:289-293 (decoding procedure), :309 (random access), :73 / :409 (two-plane rendering); definitions: DESIGN.md sections 3
// and 5; phases and vocabulary: hmlfc_render_common.cuh.
//
// A tile's decode work is a few hundred short dependent chains, so what a CTA spends on its tile is latency, and the table build (phase
// T: a few hundred instructions on one or two warps while the others wait) was a tenth of it.  Here the tables of ALL tiles are built
// first, one warp per tile, by tile_tables_kernel:
//   * the tile's footprint comes from its four CORNER pixels only.  u, v, s, t are projective functions of the pixel position; where the
//     ray direction's z is positive on the whole tile (it is affine in the position: positive at the corners is positive inside) they are
//     monotone along every pixel row and column, so every value on an edge lies between two corner values and every interior value
//     between two edge values.  The ranges get a rounding margin and are clamped to the slab; a tile with a non-positive or non-finite
//     direction at a corner, or one that spans more than 4 x 4 views, is rendered by the general path (render_tile_general);
//   * view boxes, cells, planes and accumulator offsets as in phase T of the general kernel (the same functions), written to global memory
//     (3,136 bytes per tile, most tiles use a third).
// render_tiles_kernel then loads a tile's tables and goes straight to B1 - B4; rays are set up per pixel right before the pixel's gather
// and blend (A and C fused: no per-pixel state is kept across the decode phases).  The ranges being conservative estimates, every pixel
// checks its taps against its views' boxes; one that falls outside (not seen in any test; possible in principle through rounding) is
// rendered by 16 direct sample decodes -- the result is the definition's in every case.  A tile whose tables do not fit the arena takes the
// general path (quadtree of sub-tile passes) in the same CTA.
#include "hmlfc_render_common.cuh"
#include "../../include/hmlfc.h"  // HMLFC_NOALLOC_MAX_TILES

#include <mutex>

namespace hmlfc {

namespace {

constexpr int kTile = 32;        // tile height; the width is 32 or 64 (template parameter kTW)
constexpr int kTablesWarps = 4;  // tiles per CTA of tile_tables_kernel
constexpr int kDescWords = (int)(sizeof(TileTables) / 16);
static_assert(sizeof(TileTables) % 16 == 0 && sizeof(TileHeader) == 64 && sizeof(ViewInfo) == 32 && sizeof(SlotInfo) == 64 &&
              sizeof(TileTables) == 16 * kTableHeadWords + 64 * kMaxSlots, "table layout");

// order-preserving map float -> int (no NaN)
__device__ __forceinline__ int fkey(float f) { const int k = __float_as_int(f); return k ^ ((k >> 31) & 0x7fffffff); }
__device__ __forceinline__ float fkey_inv(int k) { return __int_as_float(k ^ ((k >> 31) & 0x7fffffff)); }

// continuous (u, v, s, t) of the ray through screen point (px, py), the arithmetic of ray_from_screen without its range test;
// returns the direction's z
__device__ __forceinline__ float ray_uvst(const DevStream &S, const Camera &cam, float px, float py, float (&c)[4])
{
    const float Dx = HMLFC_ADD(HMLFC_ADD(cam.fwd[0], HMLFC_MUL(px, cam.right[0])), HMLFC_MUL(py, cam.down[0]));
    const float Dy = HMLFC_ADD(HMLFC_ADD(cam.fwd[1], HMLFC_MUL(px, cam.right[1])), HMLFC_MUL(py, cam.down[1]));
    const float Dz = HMLFC_ADD(HMLFC_ADD(cam.fwd[2], HMLFC_MUL(px, cam.right[2])), HMLFC_MUL(py, cam.down[2]));
    const float l0 = HMLFC_DIV(HMLFC_SUB(0.0f, cam.eye[2]), Dz);
    const float l1 = HMLFC_DIV(HMLFC_SUB(S.z_st, cam.eye[2]), Dz);
    const float uw = HMLFC_ADD(cam.eye[0], HMLFC_MUL(l0, Dx));
    const float vw = HMLFC_ADD(cam.eye[1], HMLFC_MUL(l0, Dy));
    const float sw = HMLFC_ADD(cam.eye[0], HMLFC_MUL(l1, Dx));
    const float tw = HMLFC_ADD(cam.eye[1], HMLFC_MUL(l1, Dy));
    c[0] = div_step(HMLFC_SUB(uw, S.uv_origin[0]), S.uv_step[0], S.uv_inv[0], S.pow2_mask & 1u);
    c[1] = div_step(HMLFC_SUB(vw, S.uv_origin[1]), S.uv_step[1], S.uv_inv[1], S.pow2_mask & 2u);
    c[2] = div_step(HMLFC_SUB(sw, S.st_origin[0]), S.st_step[0], S.st_inv[0], S.pow2_mask & 4u);
    c[3] = div_step(HMLFC_SUB(tw, S.st_origin[1]), S.st_step[1], S.st_inv[1], S.pow2_mask & 8u);
    return Dz;
}

// ---------------------------------------------------------------------------------------------------------------
// One warp per 32 x 32 tile: footprint ranges from the border pixels, then the tile's tables -> tables[tile].
__global__ void __launch_bounds__(kTablesWarps * 32)
tile_tables_kernel(const __grid_constant__ DevStream S, const Camera *__restrict__ cams, int W, int H, int tile_w, int tiles_x, int tiles_y,
                   int n_tiles, uint4 *__restrict__ tables)
{
    __shared__ TileTables stage[kTablesWarps];
    __shared__ Camera s_cam[kTablesWarps];
    __shared__ float s_aff[kTablesWarps][2][4];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int tile = blockIdx.x * kTablesWarps + warp;
    if (tile >= n_tiles) return;
    const int per_view = tiles_x * tiles_y;
    const int view = tile / per_view, tr = tile - view * per_view;
    const int ty = tr / tiles_x, tx = tr - ty * tiles_x;
    if (lane < 16) reinterpret_cast<float *>(&s_cam[warp])[lane] = reinterpret_cast<const float *>(cams + view)[lane];
    __syncwarp();
    const Camera &cam = s_cam[warp];
    if (lane < 2) camera_affine(S, cam, lane, s_aff[warp][lane]);

    // ---- corner pixels, one per lane
    const int x0 = tx * tile_w, y0 = ty * kTile;
    const int pw = min(tile_w, W - x0), ph = min(kTile, H - y0);
    int kmin[4] = {0x7fffffff, 0x7fffffff, 0x7fffffff, 0x7fffffff}, kmax[4] = {(int)0x80000000, (int)0x80000000, (int)0x80000000, (int)0x80000000};
    bool regular = true;
    if (lane < 4) {
        float c[4];
        const float Dz = ray_uvst(S, cam, ray_screen(cam.tan_half_x, W, (lane & 1) ? x0 + pw - 1 : x0),
                                  ray_screen(cam.tan_half_y, H, (lane & 2) ? y0 + ph - 1 : y0), c);
        regular = Dz > 0.0f;
#pragma unroll
        for (int a = 0; a < 4; ++a) {
            regular = regular && fabsf(c[a]) < 1e30f;  // false for NaN too
            kmin[a] = kmax[a] = fkey(c[a]);
        }
    }
    regular = __all_sync(FULL, regular);
    float fmin_[4], fmax_[4];
#pragma unroll
    for (int a = 0; a < 4; ++a) {
        fmin_[a] = fkey_inv(__reduce_min_sync(FULL, kmin[a]));
        fmax_[a] = fkey_inv(__reduce_max_sync(FULL, kmax[a]));
    }
    // integer ranges of the taps: floor(.) and floor(.) + 1, a rounding margin, clamped to the slab (closed intervals)
    const int n_ax[4] = {S.U, S.V, S.Ws, S.Ht};
    int lo[4], hi[4];
    bool empty = false;
#pragma unroll
    for (int a = 0; a < 4; ++a) {
        const float top = (float)(n_ax[a] - 1), d = (float)n_ax[a] * 5e-6f + 2e-3f;
        empty = empty || fmax_[a] < -d || fmin_[a] > top + d;
        lo[a] = (int)floorf(fminf(fmaxf(fmin_[a] - d, 0.0f), top));
        hi[a] = min((int)floorf(fminf(fmaxf(fmax_[a] + d, 0.0f), top)) + 1, n_ax[a] - 1);
    }
    TileTables &tab = stage[warp];
    TileHeader rg;
    rg.bu0 = lo[0]; rg.bv0 = lo[1]; rg.nu = hi[0] - lo[0] + 1; rg.nv = hi[1] - lo[1] + 1;
    rg.bs0 = lo[2]; rg.bs1 = hi[2]; rg.bt0 = lo[3]; rg.bt1 = hi[3];
    int status = kTileTables;
    if (!regular || rg.nu > kMaxV || rg.nv > kMaxV) status = kTileGeneral;
    else if (empty) status = kTileBackground;
    uint4 *dst = tables + (size_t)tile * kDescWords;
    if (status != kTileTables) {
        if (lane == 0) {
            TileHeader hd = rg;
            hd.nslots = hd.ncell = hd.nacc = hd.nbhmax = 0; hd.status = status; hd.m_ps = hd.m_nbh = 0u; hd._pad = 0;
            *reinterpret_cast<TileHeader *>(dst) = hd;
        }
        return;
    }
    __syncwarp();  // s_aff
    build_view_table(S, s_aff[warp], rg, tab);
    build_slot_table(S, s_aff[warp], rg, tab);
    __syncwarp();
    if (lane == 0) {
        tab.hdr.status = tab.hdr.nslots <= kMaxSlots ? kTileTables : kTileGeneral;
        tab.hdr._pad = 0;
    }
    __syncwarp();
    const int nwords = kTableHeadWords + (tab.hdr.nslots <= kMaxSlots ? 4 * tab.hdr.nslots : 0);
    const uint4 *src = reinterpret_cast<const uint4 *>(&tab);
    for (int q = lane; q < nwords; q += 32) dst[q] = src[q];
}

// the general path as a call: its registers and spills stay out of the tile kernel's own allocation (the call is rare)
template <int kArenaBytes, int kNT, int kTW, bool kSubpel = false, bool kCs = false>
__device__ __noinline__ void general_tile_call(const DevStream &S, Ctl &ctl, unsigned char *__restrict__ arena, int W, int H, uint8_t *__restrict__ out,
                                               int out_aligned, int view, int tile_x, int tile_y)
{
    // the general path's tile is kTW x (4 kNT / kTW) pixels: one call, or two for the 64 x 32 tile of 256 threads (64 x 16 each)
    constexpr int kGenTH = kNT * kPPL / kTW;
    for (int part = 0; part < kTile / kGenTH; ++part)
        render_tile_general<kArenaBytes, kNT, kTW, kSubpel, kCs>(S, ctl, arena, W, H, out, out_aligned, view, tile_x, tile_y * (kTile / kGenTH) + part);
}

// ---------------------------------------------------------------------------------------------------------------
// kTW x 32 pixels per CTA of kNT threads: 32 x 32 / 256 (4 pixels per thread), 64 x 32 / 512 (4), 64 x 32 / 256 (8)
// kSubpel: streams with half-pel motion offsets (R28; phases B2 / B3 of decode_patch); kCs: chroma-subsampled streams (R18; B1 - B3)
template <int kArenaBytes, int kMinBlocks, bool kAllPow2, int kNT, int kTW, bool kSubpel = false, bool kCs = false>
__global__ void __launch_bounds__(kNT, kMinBlocks)
render_tiles_kernel(const __grid_constant__ DevStream S, const Camera *__restrict__ cams, int W, int H, uint8_t *__restrict__ out, int out_aligned,
                    const uint4 *__restrict__ tables)
{
    constexpr int kTPR = kNT / kTile;        // threads per pixel row: thread (tid % kTPR, tid / kTPR) owns pixels x = tid % kTPR + kTPR p of its row
    constexpr int kPPT = kTW / kTPR;         // pixels per thread
    constexpr int kCPL = kTW / 32;           // tile columns per lane (screen x computed once per column)
    constexpr int kRPW = 32 / kTPR;          // pixel rows per warp
    static_assert(kTPR == 8 || kTPR == 16, "quarter warps gather for 8 neighbouring pixels");
    extern __shared__ __align__(16) unsigned char arena[];
    __shared__ Ctl ctl;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int view = blockIdx.z;
    const int ox = blockIdx.x * kTW, oy = blockIdx.y * kTile;
    const uint4 *td = tables + (size_t)((view * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x) * kDescWords;
    PHASE_MARK(-1);

    // every thread reads the header itself (one broadcast transaction per warp); meanwhile the digit table and the camera
    // (and, before the header says how many there are, one word of the tables per thread: a table has at most 200 words)
    TileHeader hd;
    static_assert(kDescWords <= 256, "one table word per thread");
    const uint4 spec = tid < kDescWords ? ldg(td + tid) : make_uint4(0u, 0u, 0u, 0u);
    {
        uint4 *h4 = reinterpret_cast<uint4 *>(&hd);
        h4[0] = ldg(td); h4[1] = ldg(td + 1); h4[2] = ldg(td + 2); h4[3] = ldg(td + 3);
    }
    for (int q = tid; q < 192; q += kNT)
        reinterpret_cast<uint32_t *>(ctl.lut)[q] = reinterpret_cast<const uint32_t *>(g_cta_digit_lut.v)[q];
    if (tid >= 64 && tid < 80) reinterpret_cast<float *>(&ctl.cam)[tid - 64] = reinterpret_cast<const float *>(cams + view)[tid - 64];
    if (tid == 32) ctl.n_rec = 0;
    const uint32_t bg = (uint32_t)S.bg[0] | ((uint32_t)S.bg[1] << 8) | ((uint32_t)S.bg[2] << 16);

    if (hd.status == kTileBackground) {
        const uint32_t rgb[4] = {bg, bg, bg, bg};
        for (int q = tid; q < kTW / kPPL * kTile; q += kNT)
            store4(out, view, W, H, ox + (q % (kTW / kPPL)) * kPPL, oy + q / (kTW / kPPL), rgb, out_aligned ? 1 : 0);
        return;
    }
    bool fast = hd.status == kTileTables && tables_fit<kArenaBytes>(hd);
    if (fast) {
        const int nwords = kTableHeadWords + 4 * hd.nslots;
        uint4 *dst = reinterpret_cast<uint4 *>(&ctl.tab);
        if (tid < nwords) dst[tid] = spec;
        for (int q = tid + kNT; q < nwords; q += kNT) dst[q] = ldg(td + q);
        uint4 *z = reinterpret_cast<uint4 *>(arena);
        const int nz = (hd.nacc + 1) >> 1;
        for (int q = tid; q < nz; q += kNT) z[q] = make_uint4(0u, 0u, 0u, 0u);
    }
    __syncthreads();
    PHASE_MARK(4);
    if (fast) fast = decode_patch<kArenaBytes, kNT, kSubpel, kCs>(S, ctl, arena, 0x7fffffff - kNT);
    if (!fast) {
        PASS_STAT(hd.status != kTileTables ? 14 : 15);
        // irregular rays, more than 4 x 4 views, or tables / records that do not fit the arena: the general path, in this CTA
        reset_ctl(ctl);
        if (tid < 2) camera_affine(S, ctl.cam, tid, ctl.aff[tid]);
        general_tile_call<kArenaBytes, kNT, kTW, kSubpel, kCs>(S, ctl, arena, W, H, out, out_aligned ? 1 : 0, view, (int)blockIdx.x, (int)blockIdx.y);
        return;
    }

    // ------------------------------------------------ A + C: per pixel, ray -> 16 taps -> gather + blend.  Thread (tid % kTPR, tid / kTPR) owns
    // pixels x = tid % kTPR + kTPR p of its row: the 8 lanes of a quarter warp gather for 8 NEIGHBOURING pixels at a time, whose taps are the
    // same few patch cells (one shared-memory wavefront per 128-bit load, where pixels 4 apart spread over 13 cells and collide)
    const Camera &cam = ctl.cam;
    const float4 *patch = reinterpret_cast<const float4 *>(arena + (((size_t)hd.nacc * 8 + 15) & ~(size_t)15));
    // screen coordinates once per column / row of the tile, shared by shuffles
    float pxl[kCPL];
#pragma unroll
    for (int j = 0; j < kCPL; ++j) pxl[j] = ray_screen(cam.tan_half_x, W, ox + 32 * j + lane);
    const float pyl = ray_screen(cam.tan_half_y, H, oy + warp * kRPW + (lane % kRPW));
    const float py = __shfl_sync(FULL, pyl, lane / kTPR);
    const int tx = tid % kTPR, y = oy + tid / kTPR;
    uint32_t rgb[kPPT];
#pragma unroll
    for (int p = 0; p < kPPT; ++p) {
        const int xr = tx + kTPR * p;  // column of the tile: computed by lane xr % 32 as its value xr / 32
        const float px = __shfl_sync(FULL, pxl[xr / 32 < kCPL ? xr / 32 : 0], xr & 31);
        rgb[p] = bg;
        if (ox + xr < W && y < H) {
            const Ray r = ray_from_screen_t<kAllPow2>(S, cam, px, py);
            if (r.hit) rgb[p] = blend_taps<true>(S, ctl, patch, tap_setup(S, r), hd.bu0, hd.bv0);
        }
    }
    PHASE_MARK(9);
    // ------------------------------------------------ stores.  Whole tiles of a 16-byte-aligned output: the tile's pixels are staged in
    // shared memory (the accumulators are dead) and leave as 16-byte stores, 6 per 96 bytes of a row, every sector written once.
    if (out_aligned == 2 && ox + kTW <= W && oy + kTile <= H) {
        constexpr int kStride = kTW + 8;  // words per staged row: the rows x columns a warp writes per step fall into 32 different banks
        constexpr int kChunks = 3 * kTW / 16;   // 16-byte chunks per row
        uint32_t *stage = reinterpret_cast<uint32_t *>(arena);
        if (hd.nacc * 8 < kTile * kStride * 4) __syncthreads();  // (CTA-uniform) the stage reaches into the patch: every pixel has gathered
#pragma unroll
        for (int p = 0; p < kPPT; ++p) stage[(tid / kTPR) * kStride + tx + kTPR * p] = rgb[p];
        __syncthreads();
        for (int q = tid; q < kChunks * kTile; q += kNT) {
            const int row = q / kChunks, k = q - row * kChunks;
            const uint32_t *src = stage + row * kStride;
            uint32_t w[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                // output word at byte b of the row's RGB stream: pixel b / 3 from its byte b % 3 on, then the next pixel
                const int b = 16 * k + 4 * j, a = (b * 21846) >> 16, r = b - 3 * a;
                const uint32_t lo = src[a], hi = a + 1 < kTW ? src[a + 1] : 0u;
                w[j] = (lo >> (8 * r)) | (hi << (24 - 8 * r));
            }
            uint8_t *o = out + 3 * (((size_t)view * H + (size_t)(oy + row)) * (size_t)W + (size_t)ox) + 16 * k;
            *reinterpret_cast<uint4 *>(o) = make_uint4(w[0], w[1], w[2], w[3]);
        }
    } else {
#pragma unroll
        for (int p = 0; p < kPPT; ++p) {
            const int x = ox + tx + kTPR * p;
            if (x < W && y < H) {
                uint8_t *o = out + 3 * (((size_t)view * H + (size_t)y) * (size_t)W + (size_t)x);
                o[0] = (uint8_t)(rgb[p] & 0xFF);
                o[1] = (uint8_t)((rgb[p] >> 8) & 0xFF);
                o[2] = (uint8_t)((rgb[p] >> 16) & 0xFF);
            }
        }
    }
    PHASE_MARK(10);
}

// 233,472 bytes of shared memory per SM, 1 KB reserved and 9.4 KB of tables per CTA
//   0: 32 x 32 tile, 256 threads, 3 CTAs x 65 KB     1: 32 x 32, 256 threads, 4 CTAs x 46 KB
//   2: 64 x 32 tile, 512 threads, 2 CTAs x 103 KB    3: 64 x 32, 256 threads (8 pixels per thread), 2 CTAs x 103 KB
//   4: 64 x 32 tile, 256 threads, 3 CTAs x 65 KB
#define HMLFC_TILES_CONFIGS(X) \
    X(0, 65 * 1024, 3, 256, 32) \
    X(1, 46 * 1024, 4, 256, 32) \
    X(2, 103 * 1024, 2, 512, 64) \
    X(3, 103 * 1024, 2, 256, 64) \
    X(4, 65 * 1024, 3, 256, 64)
constexpr int kSubpelArena = 65 * 1024;

}  // namespace

#ifdef HMLFC_PASS_STATS
extern "C" int hmlfc_debug_pass_stats_tiles(unsigned long long *out, int reset)
{
    cudaDeviceSynchronize();
    cudaMemcpyFromSymbol(out, g_pass_stats, sizeof(g_pass_stats));
    if (reset) { unsigned long long z[64] = {}; cudaMemcpyToSymbol(g_pass_stats, z, sizeof(z)); }
    return 0;
}
#endif

size_t render_tiles_scratch_bytes(int n_views, int W, int H)
{
    const size_t n_tiles = (size_t)n_views * (size_t)((W + kTile - 1) / kTile) * (size_t)((H + kTile - 1) / kTile);  // enough for either width
    return n_tiles * sizeof(TileTables);
}

cudaError_t configure_render_tiles()
{
    cudaError_t e = cudaSuccess;
#define X(id, arena, minb, nt, tw) \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(render_tiles_kernel<arena, minb, false, nt, tw>, cudaFuncAttributeMaxDynamicSharedMemorySize, arena); \
    if (e == cudaSuccess) e = cudaFuncSetAttribute(render_tiles_kernel<arena, minb, true, nt, tw>, cudaFuncAttributeMaxDynamicSharedMemorySize, arena);
    HMLFC_TILES_CONFIGS(X)
#undef X
    // half-pel streams: configuration 0 only
    if (e == cudaSuccess) e = cudaFuncSetAttribute(render_tiles_kernel<kSubpelArena, 3, false, 256, 32, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSubpelArena);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(render_tiles_kernel<kSubpelArena, 3, true, 256, 32, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSubpelArena);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(render_tiles_kernel<kSubpelArena, 3, false, 256, 32, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSubpelArena);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(render_tiles_kernel<kSubpelArena, 3, true, 256, 32, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSubpelArena);
    return e;
}

cudaError_t launch_render_tiles(const DevStream &S, const Camera *d_cams, int n_views, int W, int H, uint8_t *d_out, void *d_scratch,
                                cudaStream_t st, int *n_launches, int config)
{
    if (n_views == 0) return cudaSuccess;
    if (S.B != 4 || !d_scratch) return cudaErrorInvalidValue;
    const int tile_w = config >= 2 ? 64 : 32;
    const int tiles_x = (W + tile_w - 1) / tile_w, tiles_y = (H + kTile - 1) / kTile;
    const long long n_tiles_ll = (long long)n_views * tiles_x * tiles_y;
    if (tiles_y > 65535 || tiles_x > 65535 || n_tiles_ll > 0x3fffffffLL) return cudaErrorInvalidValue;
    const int n_tiles = (int)n_tiles_ll;
    uint4 *tables = reinterpret_cast<uint4 *>(d_scratch);
    // 2: rows of tiles start at 16-byte boundaries (staged 16-byte stores), 1: 4-pixel groups at 4-byte boundaries, 0: byte stores
    const int aligned = ((reinterpret_cast<uintptr_t>(d_out) & 15u) == 0 && (W % 16) == 0) ? 2 :
                        ((reinterpret_cast<uintptr_t>(d_out) & 3u) == 0 && (W % 4) == 0) ? 1 : 0;
    tile_tables_kernel<<<(unsigned)((n_tiles + kTablesWarps - 1) / kTablesWarps), kTablesWarps * 32, 0, st>>>(S, d_cams, W, H, tile_w, tiles_x, tiles_y,
                                                                                                          n_tiles, tables);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    dim3 grid((unsigned)tiles_x, (unsigned)tiles_y, (unsigned)n_views);
    if (S.cs) {  // chroma-subsampled streams: 32 x 32 tiles, 3 CTAs per SM whatever the configuration asked for
        if (S.sp || config >= 2) return cudaErrorInvalidValue;  // (both at once: the caller routes to the per-sample kernel)
        if (S.pow2_mask == 15u) render_tiles_kernel<kSubpelArena, 3, true, 256, 32, false, true><<<grid, 256, kSubpelArena, st>>>(S, d_cams, W, H, d_out, aligned, tables);
        else render_tiles_kernel<kSubpelArena, 3, false, 256, 32, false, true><<<grid, 256, kSubpelArena, st>>>(S, d_cams, W, H, d_out, aligned, tables);
    } else if (S.sp) {  // half-pel streams: likewise
        if (S.mv_off > 127 || config >= 2) return cudaErrorInvalidValue;  // (the records pack an offset in 8 bits; the caller routes)
        if (S.pow2_mask == 15u) render_tiles_kernel<kSubpelArena, 3, true, 256, 32, true><<<grid, 256, kSubpelArena, st>>>(S, d_cams, W, H, d_out, aligned, tables);
        else render_tiles_kernel<kSubpelArena, 3, false, 256, 32, true><<<grid, 256, kSubpelArena, st>>>(S, d_cams, W, H, d_out, aligned, tables);
    } else {
#define X(id, arena, minb, nt, tw) \
    if (config == id) { \
        if (S.pow2_mask == 15u) render_tiles_kernel<arena, minb, true, nt, tw><<<grid, nt, arena, st>>>(S, d_cams, W, H, d_out, aligned, tables); \
        else render_tiles_kernel<arena, minb, false, nt, tw><<<grid, nt, arena, st>>>(S, d_cams, W, H, d_out, aligned, tables); \
    }
    HMLFC_TILES_CONFIGS(X)
#undef X
    }
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    if (n_launches) *n_launches += 2;
    return cudaSuccess;
}

// ---------------------------------------------------------------------------------------------------------------
// hmlfc_render_noalloc: the tile path with its tables in a buffer that exists from the moment the library is loaded, for callers that
// cannot allocate (CUDA graph capture, tight serving loops).  The buffer is a file-scope __device__ array: every GPU that loads the
// library holds its kNoAllocMaxTiles x 3,200 bytes (13.1 MB) until the process exits.  In host code the array's NAME is a host-side
// stand-in, not a device address; the device address comes from cudaGetSymbolAddress, asked for once per device at set-up
// (configure_render_tiles_noalloc, called by hmlfc_load with its device current) and passed to the kernels.
// Every call on a device shares the array.  Nothing in it has to start at zero (tile_tables_kernel writes every word the render kernel
// reads: the header of every tile, the slot words the header counts), so a call leaves the previous call's contents to be overwritten;
// two calls that overlap on the GPU (different streams, no dependency) RACE on it.
constexpr int kNoAllocMaxTiles = HMLFC_NOALLOC_MAX_TILES;
constexpr int kNoAllocMaxDevices = 64;
static __device__ __align__(256) unsigned char g_noalloc_tables[(size_t)kNoAllocMaxTiles * sizeof(TileTables)];
static void *g_noalloc_ptr[kNoAllocMaxDevices];  // device address of g_noalloc_tables on device i (null: not set up there)
static std::mutex g_noalloc_mutex;

cudaError_t configure_render_tiles_noalloc()
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kNoAllocMaxDevices) return cudaSuccess;  // the entry point will say that this device was not set up
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (g_noalloc_ptr[dev]) return cudaSuccess;
    void *ptr = nullptr;
    if ((e = cudaGetSymbolAddress(&ptr, g_noalloc_tables)) != cudaSuccess) return e;
    g_noalloc_ptr[dev] = ptr;
    return cudaSuccess;
}

// *too_large: the batch has more tiles than the buffer holds (nothing was launched).  Calls no allocating routine.
cudaError_t launch_render_tiles_noalloc(const DevStream &S, const Camera *d_cams, int n_views, int W, int H, uint8_t *d_out, cudaStream_t st,
                                        int *n_launches, int config, bool *too_large)
{
    *too_large = false;
    if (n_views == 0) return cudaSuccess;
    const int tile_w = config >= 2 ? 64 : 32;
    const long long n_tiles = (long long)n_views * ((W + tile_w - 1) / tile_w) * ((H + kTile - 1) / kTile);
    if (n_tiles > kNoAllocMaxTiles) { *too_large = true; return cudaSuccess; }
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    void *ptr = nullptr;
    if (dev >= 0 && dev < kNoAllocMaxDevices) {
        std::lock_guard<std::mutex> lock(g_noalloc_mutex);
        ptr = g_noalloc_ptr[dev];
    }
    if (!ptr) return cudaErrorInvalidDevice;  // no hmlfc_load ran with this device current
    return launch_render_tiles(S, d_cams, n_views, W, H, d_out, ptr, st, n_launches, config);
}


}  // namespace hmlfc
