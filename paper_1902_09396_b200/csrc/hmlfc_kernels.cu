// HMLFC kernels for sm_100a: random-access decode, per-pixel fused render, footprint accounting.
#include "hmlfc_kernels.cuh"

namespace hmlfc {

namespace {

constexpr int kDecodeThreads = 256;

// Write one RGB triple per lane.  When the warp's 32 pixels are contiguous, 4-byte aligned and all
// present, the 96 bytes go through shared memory and leave as 24 coalesced 32-bit stores.
__device__ __forceinline__ void store_rgb_warp(uint8_t *out_warp_base, bool warp_full_aligned, bool valid, uint32_t rgb,
                                               uint32_t *stage /* 24 words of this warp */)
{
    const int lane = threadIdx.x & 31;
    if (warp_full_aligned) {
        uint8_t *sb = reinterpret_cast<uint8_t *>(stage);
        sb[3 * lane + 0] = (uint8_t)(rgb & 0xFF);
        sb[3 * lane + 1] = (uint8_t)((rgb >> 8) & 0xFF);
        sb[3 * lane + 2] = (uint8_t)((rgb >> 16) & 0xFF);
        __syncwarp();
        if (lane < 24) reinterpret_cast<uint32_t *>(out_warp_base)[lane] = stage[lane];
        __syncwarp();
    } else if (valid) {
        uint8_t *o = out_warp_base + 3 * lane;
        o[0] = (uint8_t)(rgb & 0xFF);
        o[1] = (uint8_t)((rgb >> 8) & 0xFF);
        o[2] = (uint8_t)((rgb >> 16) & 0xFF);
    }
}

// ---------------------------------------------------------------- hmlfc_decode
// One thread per coordinate: a pure gather.  PAPER.md:309 "parallel decompression of different
// pixel values from the compressed stream".
__global__ void __launch_bounds__(kDecodeThreads)
decode_kernel(const DevStream S, const int4 *__restrict__ coords, long long n, uint8_t *__restrict__ out,
              unsigned long long *oob, int out_aligned)
{
    __shared__ uint32_t stage[kDecodeThreads / 32][24];
    const long long i = (long long)blockIdx.x * kDecodeThreads + threadIdx.x;
    const bool valid = i < n;
    uint32_t rgb = 0;
    if (valid) {
        int4 q = __ldg(coords + i);
        if ((unsigned)q.x < (unsigned)S.U && (unsigned)q.y < (unsigned)S.V && (unsigned)q.z < (unsigned)S.Ws &&
            (unsigned)q.w < (unsigned)S.Ht)
            rgb = decode_rgb8(S, q.x, q.y, q.z, q.w);
        else
            atomicAdd(oob, 1ull);
    }
    const long long wbase = i - (threadIdx.x & 31);
    store_rgb_warp(out + 3 * wbase, out_aligned && (wbase + 32 <= n), valid, rgb, stage[threadIdx.x >> 5]);
}

// hmlfc_decode_views / hmlfc_decode_blocks with one thread per pixel, the coordinates generated here (kBlocks: sample i is pixel
// i mod B^2 of block blocks[i / B^2] = (u, v, bx, by); else pixel i mod (Ws Ht) of view views[i / (Ws Ht)] = (u, v)).  The path of
// chroma-subsampled streams (R18), which the block-row and warp-cooperative kernels do not read.
template <bool kBlocks>
__global__ void __launch_bounds__(kDecodeThreads)
decode_dense_kernel(const DevStream S, const int32_t *__restrict__ list, long long n, uint8_t *__restrict__ out, unsigned long long *oob,
                    int out_aligned)
{
    __shared__ uint32_t stage[kDecodeThreads / 32][24];
    const long long i = (long long)blockIdx.x * kDecodeThreads + threadIdx.x;
    const bool valid = i < n;
    uint32_t rgb = 0;
    if (valid) {
        int u, v, x, y;
        bool ok;
        if (kBlocks) {
            const int bb = S.B * S.B;
            const long long blk = i / bb;
            const int k = (int)(i - blk * bb), ky = k >> S.logB;
            const int4 q = __ldg(reinterpret_cast<const int4 *>(list) + blk);
            u = q.x; v = q.y; x = q.z * S.B + (k - (ky << S.logB)); y = q.w * S.B + ky;
            ok = (unsigned)q.z < (unsigned)S.nbx && (unsigned)q.w < (unsigned)S.nby;
        } else {
            const long long npx = (long long)S.Ws * S.Ht;
            const long long view = i / npx;
            const int pix = (int)(i - view * npx);
            const int2 uv = __ldg(reinterpret_cast<const int2 *>(list) + view);
            u = uv.x; v = uv.y; y = pix / S.Ws; x = pix - y * S.Ws;
            ok = true;
        }
        if (ok && (unsigned)u < (unsigned)S.U && (unsigned)v < (unsigned)S.V) rgb = decode_rgb8(S, u, v, x, y);
        else atomicAdd(oob, 1ull);
    }
    const long long wbase = i - (threadIdx.x & 31);
    store_rgb_warp(out + 3 * wbase, out_aligned && (wbase + 32 <= n), valid, rgb, stage[threadIdx.x >> 5]);
}

// ---------------------------------------------------------------- hmlfc_render, one thread per output pixel
// Ray set-up -> 16 taps -> 16 independent sample decodes -> quadrilinear blend -> RGB8 store.
constexpr int kPixTx = 32, kPixTy = 8;

__device__ __forceinline__ void blend_add(float acc[3], float w, uint32_t rgb)
{
    acc[0] = fmaf(w, (float)(rgb & 0xFF), acc[0]);
    acc[1] = fmaf(w, (float)((rgb >> 8) & 0xFF), acc[1]);
    acc[2] = fmaf(w, (float)((rgb >> 16) & 0xFF), acc[2]);
}

__device__ __forceinline__ uint32_t round_rgb(const float acc[3])
{
    // out = floor(x + 0.5), x in [0,255]
    uint32_t r = (uint32_t)min(max(__float2int_rd(acc[0] + 0.5f), 0), 255);
    uint32_t g = (uint32_t)min(max(__float2int_rd(acc[1] + 0.5f), 0), 255);
    uint32_t b = (uint32_t)min(max(__float2int_rd(acc[2] + 0.5f), 0), 255);
    return r | (g << 8) | (b << 16);
}

__global__ void __launch_bounds__(kPixTx *kPixTy)
render_pixel_kernel(const DevStream S, const Camera *__restrict__ cams, int W, int H, uint8_t *__restrict__ out,
                    int out_aligned)
{
    __shared__ uint32_t stage[kPixTy][24];
    const int i = blockIdx.x * kPixTx + threadIdx.x;
    const int j = blockIdx.y * kPixTy + threadIdx.y;
    const int view = blockIdx.z;
    const bool valid = i < W && j < H;
    uint32_t rgb = (uint32_t)S.bg[0] | ((uint32_t)S.bg[1] << 8) | ((uint32_t)S.bg[2] << 16);
    if (valid) {
        const Camera cam = cams[view];
        Ray r = ray_setup(S, cam, W, H, i, j);
        if (r.hit) {
            Taps k = tap_setup(S, r);
            float acc[3] = {0.f, 0.f, 0.f};
#pragma unroll 1
            for (int a = 0; a < 4; ++a) {
                const int uu = (a & 1) ? k.u1 : k.u0, vv = (a & 2) ? k.v1 : k.v0;
                const float wuv = ((a & 1) ? k.fu : 1.0f - k.fu) * ((a & 2) ? k.fv : 1.0f - k.fv);
                float C[3] = {0.f, 0.f, 0.f};
#pragma unroll 1
                for (int b = 0; b < 4; ++b) {
                    const int ss = (b & 1) ? k.s1 : k.s0, tt = (b & 2) ? k.t1 : k.t0;
                    const float wst = ((b & 1) ? k.fs : 1.0f - k.fs) * ((b & 2) ? k.ft : 1.0f - k.ft);
                    blend_add(C, wst, decode_rgb8(S, uu, vv, ss, tt));
                }
                acc[0] = fmaf(wuv, C[0], acc[0]);
                acc[1] = fmaf(wuv, C[1], acc[1]);
                acc[2] = fmaf(wuv, C[2], acc[2]);
            }
            rgb = round_rgb(acc);
        }
    }
    const int i0 = blockIdx.x * kPixTx;
    uint8_t *row = out + 3 * (((size_t)view * H + (size_t)min(j, H - 1)) * (size_t)W + (size_t)i0);
    store_rgb_warp(row, out_aligned && (i0 + 32 <= W) && (j < H), valid, rgb, stage[threadIdx.y]);
}

// ---------------------------------------------------------------- footprint (measurement aid)
__device__ __forceinline__ void mark_bit(uint32_t *bits, size_t idx)
{
    const uint32_t m = 1u << (idx & 31);
    uint32_t *w = bits + (idx >> 5);
    if (!(*(volatile uint32_t *)w & m)) atomicOr(w, m);
}

__device__ void touch_sample(const DevStream &S, FootprintMarks mk, int u, int v, int x, int y)
{
    const int h = S.h;
    mark_bit(mk.rkv, ((size_t)((v >> h) * S.UH + (u >> h)) * (size_t)S.Ht + (size_t)y) * (size_t)S.Ws + (size_t)x);
    const int b = (y >> S.logB) * S.nbx + (x >> S.logB);
    const uint32_t bit = 1u << (b & 31);
    for (int L = S.lmin; L < h; ++L) {
        const int pu = u >> L, pv = v >> L;
        const LevelDesc lv = S.lev[L];
        const uint32_t base = lv.pc_base + (uint32_t)(pv * lv.UL + pu) * 3u;
        const uint32_t rbase = lv.pc_base + (uint32_t)((pv & ~1) * lv.UL + (pu & ~1)) * 3u;
        for (int c = 0; c < 3; ++c) {
            mark_bit(mk.blk, (size_t)(base + c) * (size_t)S.nblk + (size_t)b);
            if (!((pu | pv) & 1)) continue;
            uint4 d = ldg(S.pc + base + c);
            uint4 fr = ldg(S.flagrec + d.x + 4u * (uint32_t)(b >> 5));
            if (!(fr.z & bit)) continue;
            uint32_t rec = bise_decode_at(S.mv + d.z, fr.w + popc(fr.z & (bit - 1u)), S.mv_layout, S.mv_m);
            int mode, dx, dy;
            mv_unpack(S, rec, mode, dx, dy);
            const int rx = x + dx, ry = y + dy;
            if ((unsigned)rx < (unsigned)S.Ws && (unsigned)ry < (unsigned)S.Ht)
                mark_bit(mk.blk, (size_t)(rbase + c) * (size_t)S.nblk + (size_t)((ry >> S.logB) * S.nbx + (rx >> S.logB)));
        }
    }
}

__global__ void footprint_render_kernel(const DevStream S, const Camera *__restrict__ cams, int W, int H, FootprintMarks mk)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    if (i >= W || j >= H) return;
    const Camera cam = cams[blockIdx.z];
    Ray r = ray_setup(S, cam, W, H, i, j);
    if (!r.hit) return;
    Taps k = tap_setup(S, r);
    for (int a = 0; a < 16; ++a)
        touch_sample(S, mk, (a & 1) ? k.u1 : k.u0, (a & 2) ? k.v1 : k.v0, (a & 4) ? k.s1 : k.s0, (a & 8) ? k.t1 : k.t0);
}

__global__ void footprint_decode_kernel(const DevStream S, const int4 *__restrict__ coords, long long n, FootprintMarks mk)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int4 q = __ldg(coords + i);
    if ((unsigned)q.x < (unsigned)S.U && (unsigned)q.y < (unsigned)S.V && (unsigned)q.z < (unsigned)S.Ws &&
        (unsigned)q.w < (unsigned)S.Ht)
        touch_sample(S, mk, q.x, q.y, q.z, q.w);
}

// one thread per (plane-channel, 32-block group): reduce the marks to bit counts
__global__ void footprint_reduce_blocks_kernel(const DevStream S, unsigned long long n_groups_total,
                                               const uint32_t *__restrict__ bits15, uint32_t mv_bits15, FootprintMarks mk,
                                               FootprintTotals *tot)
{
    const unsigned long long gi = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long blocks = 0, flag_bits = 0, pay = 0, mvb = 0;
    if (gi < n_groups_total) {
        const uint32_t k = (uint32_t)(gi / (unsigned)S.fgroups), g = (uint32_t)(gi % (unsigned)S.fgroups);
        // marks are indexed by k*nblk + b: gather this group's 32 bits (nblk need not be a multiple of 32)
        uint32_t marks = 0;
        for (int j = 0; j < 32; ++j) {
            const int b = (int)g * 32 + j;
            if (b >= S.nblk) break;
            const size_t idx = (size_t)k * (size_t)S.nblk + (size_t)b;
            marks |= ((mk.blk[idx >> 5] >> (idx & 31)) & 1u) << j;
        }
        if (marks) {
            uint4 d = ldg(S.pc + k);
            uint4 fr = ldg(S.flagrec + d.x + 4u * g);
            const bool isp = pc_is_pred(d.w);
            blocks = popc(marks);
            flag_bits = blocks * (isp ? 2u : 1u);
            pay = (unsigned long long)popc(marks & fr.x) * bits15[k] * (unsigned)(S.B * S.B);
            if (isp) mvb = (unsigned long long)popc(marks & fr.z) * mv_bits15;
        }
    }
    // block-level reduction through warp shuffles + one atomic per warp
    for (int o = 16; o > 0; o >>= 1) {
        blocks += __shfl_down_sync(0xffffffffu, blocks, o);
        flag_bits += __shfl_down_sync(0xffffffffu, flag_bits, o);
        pay += __shfl_down_sync(0xffffffffu, pay, o);
        mvb += __shfl_down_sync(0xffffffffu, mvb, o);
    }
    if ((threadIdx.x & 31) == 0 && blocks) {
        atomicAdd(&tot->blocks, blocks);
        atomicAdd(&tot->flag_bits, flag_bits);
        atomicAdd(&tot->payload_bits15, pay);
        atomicAdd(&tot->mv_bits15, mvb);
    }
}

__global__ void footprint_reduce_rkv_kernel(const uint32_t *__restrict__ marks, unsigned long long n_words, FootprintTotals *tot)
{
    unsigned long long cnt = 0;
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_words;
         i += (unsigned long long)gridDim.x * blockDim.x)
        cnt += popc(marks[i]);
    for (int o = 16; o > 0; o >>= 1) cnt += __shfl_down_sync(0xffffffffu, cnt, o);
    if ((threadIdx.x & 31) == 0 && cnt) atomicAdd(&tot->rkv_samples, cnt);
}

}  // namespace

// ---------------------------------------------------------------- launchers
cudaError_t launch_decode(const DevStream &S, const int32_t *d_coords, int64_t n, uint8_t *d_out,
                          unsigned long long *d_oob, cudaStream_t st, int *n_launches)
{
    if (n == 0) return cudaSuccess;
    const long long blocks = (n + kDecodeThreads - 1) / kDecodeThreads;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidValue;
    const int aligned = ((reinterpret_cast<uintptr_t>(d_out) & 3u) == 0) ? 1 : 0;
    decode_kernel<<<(unsigned)blocks, kDecodeThreads, 0, st>>>(S, reinterpret_cast<const int4 *>(d_coords), (long long)n, d_out,
                                                                d_oob, aligned);
    if (n_launches) *n_launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_decode_dense(const DevStream &S, const int32_t *d_list, int64_t n_items, bool blocks, uint8_t *d_out,
                                unsigned long long *d_oob, cudaStream_t st, int *n_launches)
{
    if (n_items == 0) return cudaSuccess;
    const long long n = (long long)n_items * (blocks ? (long long)S.B * S.B : (long long)S.Ws * S.Ht);
    const long long ctas = (n + kDecodeThreads - 1) / kDecodeThreads;
    if (ctas > 0x7fffffffLL) return cudaErrorInvalidValue;
    const int aligned = ((reinterpret_cast<uintptr_t>(d_out) & 3u) == 0) ? 1 : 0;
    if (blocks) decode_dense_kernel<true><<<(unsigned)ctas, kDecodeThreads, 0, st>>>(S, d_list, n, d_out, d_oob, aligned);
    else decode_dense_kernel<false><<<(unsigned)ctas, kDecodeThreads, 0, st>>>(S, d_list, n, d_out, d_oob, aligned);
    if (n_launches) *n_launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_render_pixel(const DevStream &S, const Camera *d_cams, int n_views, int W, int H, uint8_t *d_out,
                                cudaStream_t st, int *n_launches)
{
    if (n_views == 0) return cudaSuccess;
    dim3 block(kPixTx, kPixTy), grid((W + kPixTx - 1) / kPixTx, (H + kPixTy - 1) / kPixTy, n_views);
    const int aligned = ((reinterpret_cast<uintptr_t>(d_out) & 3u) == 0 && (W % 4) == 0) ? 1 : 0;
    render_pixel_kernel<<<grid, block, 0, st>>>(S, d_cams, W, H, d_out, aligned);
    if (n_launches) *n_launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_footprint_render(const DevStream &S, const Camera *d_cams, int n_views, int W, int H,
                                    FootprintMarks marks, cudaStream_t st)
{
    if (n_views == 0) return cudaSuccess;
    dim3 block(32, 8), grid((W + 31) / 32, (H + 7) / 8, n_views);
    footprint_render_kernel<<<grid, block, 0, st>>>(S, d_cams, W, H, marks);
    return cudaGetLastError();
}

cudaError_t launch_footprint_decode(const DevStream &S, const int32_t *d_coords, int64_t n, FootprintMarks marks,
                                    cudaStream_t st)
{
    if (n == 0) return cudaSuccess;
    const long long blocks = (n + 255) / 256;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidValue;
    footprint_decode_kernel<<<(unsigned)blocks, 256, 0, st>>>(S, reinterpret_cast<const int4 *>(d_coords), (long long)n, marks);
    return cudaGetLastError();
}

cudaError_t launch_footprint_reduce(const DevStream &S, uint64_t n_pc, const uint32_t *d_bits15, uint32_t mv_bits15,
                                    FootprintMarks marks, FootprintTotals *d_totals, cudaStream_t st)
{
    const unsigned long long n_groups = (unsigned long long)n_pc * (unsigned long long)S.fgroups;
    const unsigned long long blocks = (n_groups + 255) / 256;
    if (blocks > 0x7fffffffULL) return cudaErrorInvalidValue;
    footprint_reduce_blocks_kernel<<<(unsigned)blocks, 256, 0, st>>>(S, n_groups, d_bits15, mv_bits15, marks, d_totals);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    const unsigned long long n_words = ((unsigned long long)S.UH * S.VH * S.Ht * S.Ws + 31) / 32;
    footprint_reduce_rkv_kernel<<<1024, 256, 0, st>>>(marks.rkv, n_words, d_totals);
    return cudaGetLastError();
}

}  // namespace hmlfc
