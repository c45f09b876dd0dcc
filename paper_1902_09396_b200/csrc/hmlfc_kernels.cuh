// Launchers of the HMLFC kernels (definitions in hmlfc_kernels.cu, hmlfc_decode_queue.cu, hmlfc_render_warp.cu, hmlfc_render_cta.cu).
#pragma once

#include "hmlfc_device.cuh"

namespace hmlfc {

// Device scratch from a library-owned stream-ordered pool of the current device (cudaMallocFromPoolAsync): after the first call the pool
// serves the buffers without going to the driver, and frees do not synchronise the device.  scratch_pool_trim returns the memory.
cudaError_t scratch_pool(cudaMemPool_t *out);
cudaError_t scratch_pool_trim();

// marks written by the footprint kernels
struct FootprintMarks {
    uint32_t *blk;  // [n_pc * nblk] bits
    uint32_t *rkv;  // [UH * VH * Ht * Ws] bits
};

struct FootprintTotals {
    unsigned long long blocks, flag_bits, payload_bits15, mv_bits15, rkv_samples;
};

cudaError_t launch_decode(const DevStream &S, const int32_t *d_coords, int64_t n, uint8_t *d_out,
                          unsigned long long *d_oob, cudaStream_t st, int *n_launches);
// warp-cooperative decode (hmlfc_decode_queue.cu): same result as launch_decode
// mode: 0 = flag records and descriptors up front (eager); 1 = one flag sector per level, tasks fetch descriptor and rank (lazy); 2 = the
// block records (S.brec); -1 = block records where the stream has them, else lazy / eager by S.l2_resident
cudaError_t launch_decode_queue(const DevStream &S, const int32_t *d_coords, int64_t n, uint8_t *d_out,
                                unsigned long long *d_oob, cudaStream_t st, int *n_launches, int mode = -1);
cudaError_t configure_decode_queue();
// whole views: d_views = int32 [n_views][2] = (u, v); d_out = uint8 [n_views][Ht][Ws][3]; coordinates are generated in the kernel
cudaError_t launch_decode_views(const DevStream &S, const int32_t *d_views, int64_t n_views, uint8_t *d_out, unsigned long long *d_oob,
                                cudaStream_t st, int *n_launches);
// the same for B = 4 streams: one lane per block-row segment (hmlfc_render_cta.cu)
cudaError_t launch_decode_rows(const DevStream &S, const int32_t *d_views, int64_t n_views, uint8_t *d_out, unsigned long long *d_oob,
                               cudaStream_t st, int *n_launches);
// whole B x B blocks: d_blocks = int32 [n][4] = (u, v, bx, by); d_out = uint8 [n][B][B][3]; lane per pixel (any B) / per block row (B = 4)
cudaError_t launch_decode_blocks(const DevStream &S, const int32_t *d_blocks, int64_t n_blocks, uint8_t *d_out, unsigned long long *d_oob,
                                 cudaStream_t st, int *n_launches);
cudaError_t launch_decode_block_rows(const DevStream &S, const int32_t *d_blocks, int64_t n_blocks, uint8_t *d_out, unsigned long long *d_oob,
                                     cudaStream_t st, int *n_launches);
// one thread per pixel of whole views (d_list = int32 [n][2]) or whole blocks (int32 [n][4]): any stream, incl. chroma-subsampled ones
cudaError_t launch_decode_dense(const DevStream &S, const int32_t *d_list, int64_t n_items, bool blocks, uint8_t *d_out,
                                unsigned long long *d_oob, cudaStream_t st, int *n_launches);
cudaError_t launch_render_pixel(const DevStream &S, const Camera *d_cams, int n_views, int W, int H, uint8_t *d_out,
                                cudaStream_t st, int *n_launches);
// shape 0: 16 x 8 tiles (4 pixels per lane), 1: 8 x 8 tiles (2 pixels per lane)
cudaError_t launch_render_warp(const DevStream &S, const Camera *d_cams, int n_views, int W, int H, uint8_t *d_out, cudaStream_t st,
                               int *n_launches, int shape);
cudaError_t configure_render_warp();
// Fused render kernels for B = 4 streams (return cudaErrorInvalidValue otherwise).
// launch_render_cta (hmlfc_render_cta.cu): tables built inside the CTA, quadtree of sub-tile passes.  config: 0 = 256 threads, 32 x 32
// tile, 3 CTAs x 66 KB per SM, 1 = 2 CTAs x 104 KB, 2 = 4 CTAs x 47 KB, 3 = 1024 threads, 64 x 64 tile, 4 = 512 threads, 64 x 32 tile,
// -1 = chosen from the output and light-field sizes.
cudaError_t launch_render_cta(const DevStream &S, const Camera *d_cams, int n_views, int W, int H, uint8_t *d_out, cudaStream_t st,
                              int *n_launches, int config);
// launch_render_tiles (hmlfc_render_tiles.cu): tile tables built by a kernel of their own from the tiles' border rays, one pass per 32 x 32
// tile (a tile that does not fit takes the general kernel's path in its CTA).  d_scratch: render_tiles_scratch_bytes() bytes of device
// memory for the tables (contents irrelevant before, undefined after).  config: 0 / 1 = 32 x 32 tiles, 3 / 4 CTAs per SM; 2 = 64 x 32 tiles, 512 threads;
// 3 / 4 = 64 x 32 tiles, 256 threads (8 pixels per thread), 2 / 3 CTAs per SM.
size_t render_tiles_scratch_bytes(int n_views, int W, int H);

// hmlfc_load: block records of the uploaded stream S (S.pb set) -> d_brec (zeroed), hmlfc_repack.cu
cudaError_t launch_repack(const DevStream &S, uint64_t n_planes, uint32_t *d_brec, cudaStream_t st);
cudaError_t launch_render_tiles(const DevStream &S, const Camera *d_cams, int n_views, int W, int H, uint8_t *d_out, void *d_scratch,
                                cudaStream_t st, int *n_launches, int config);
// the same with the tables in the library's static device buffer (hmlfc_render_noalloc; at most HMLFC_NOALLOC_MAX_TILES tiles per call):
// set-up once per device (by hmlfc_load), then launches that allocate nothing
cudaError_t configure_render_tiles_noalloc();
cudaError_t launch_render_tiles_noalloc(const DevStream &S, const Camera *d_cams, int n_views, int W, int H, uint8_t *d_out, cudaStream_t st,
                                        int *n_launches, int config, bool *too_large);
cudaError_t configure_render_tiles();
cudaError_t configure_render_cta();
cudaError_t launch_footprint_render(const DevStream &S, const Camera *d_cams, int n_views, int W, int H,
                                    FootprintMarks marks, cudaStream_t st);
cudaError_t launch_footprint_decode(const DevStream &S, const int32_t *d_coords, int64_t n, FootprintMarks marks,
                                    cudaStream_t st);
// bits15[k] = BISE bits per value of plane-channel k in units of 1/15 bit
cudaError_t launch_footprint_reduce(const DevStream &S, uint64_t n_pc, const uint32_t *d_bits15, uint32_t mv_bits15,
                                    FootprintMarks marks, FootprintTotals *d_totals, cudaStream_t st);

}  // namespace hmlfc
