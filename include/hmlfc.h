/*
 * hmlfc.h -- C ABI of the B200-native HMLFC decode + render library (libhmlfc_b200.so).
 *
 * The hot path of "HMLFC: Hierarchical Motion-Compensated Light Field Compression for
 * Interactive Rendering" (arXiv 1902.09396): random-access per-pixel decoding of the
 * hierarchical, phase-shifted motion-compensated representation (section
 * 4.8), fused with two-plane (u,v,s,t) novel-view rendering.
 * Every step runs in hand-written CUDA kernels for sm_100a; there is no CPU fallback.
 *
 * Conventions
 *   - (u,v) = camera-grid index, U x V views; (s,t) = pixel column/row inside a view, Ws x Ht.
 *   - All functions return 0 on success or a negative HMLFC_E_* code; no exceptions cross the ABI.
 *   - Pointers named h_* are HOST pointers, d_* are DEVICE pointers on the device that was
 *     current when hmlfc_load() ran.  cuda_stream is a cudaStream_t passed as void* (NULL = the
 *     legacy default stream).
 *   - decode / render / footprint only ENQUEUE work on cuda_stream and return without
 *     synchronising; the *_host variants synchronise before returning.
 *   - The handle is immutable after load apart from its counters; concurrent launches on
 *     different streams are legal (the out-of-range counter is shared and atomic).
 */
#ifndef HMLFC_H
#define HMLFC_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    HMLFC_OK = 0,
    HMLFC_E_MAGIC = -1,        /* stream does not start with "HMLF"                          */
    HMLFC_E_TRUNCATED = -2,    /* fewer bytes than the header / directory say                */
    HMLFC_E_VERSION = -3,      /* stream version is not 1                                    */
    HMLFC_E_INVALID = -4,      /* null pointer, n < 0, W/H <= 0, ...                          */
    HMLFC_E_UNSUPPORTED = -5,  /* B not in {2,4,8} or B does not divide Ws/Ht, chroma         */
                               /* subsampling set, RKV codec != raw, height > 8              */
    HMLFC_E_CORRUPT = -6,      /* directory inconsistent with the section sizes              */
    HMLFC_E_NOMEM = -7,        /* host or device allocation failed                           */
    HMLFC_E_CUDA = -8,         /* a CUDA runtime call failed (see hmlfc_last_cuda_error)     */
    HMLFC_E_LIMIT = -9         /* the request exceeds a fixed capacity (hmlfc_render_noalloc) */
};

typedef struct hmlfc_handle hmlfc_handle; /* opaque; owns every device allocation */

/* Stream parameters (header of the compressed stream) and the sizes of its device form. */
typedef struct {
    int32_t U, V, Ws, Ht;
    int32_t height;            /* tree height h ("tree height")              */
    int32_t block;             /* block size B                                            */
    int32_t window;            /* search window W: motion vectors lie in [-W, W]^2        */
    int32_t tau_ref, tau_res;  /* the encoder's two block thresholds       */
    float uv_origin[2], uv_step[2], st_origin[2], st_step[2], z_st; /* light slab geometry */
    uint8_t background[3];     /* colour of rays that miss the slab                       */
    uint8_t _pad;
    uint64_t stream_bytes;     /* length of the serialized stream                         */
    uint64_t device_bytes;     /* bytes resident in HBM after load (all tables)           */
    uint64_t n_plane_channels; /* SRV plane-channels in the tree                          */
} hmlfc_info_t;

/* One output camera: a ray basis, not necessarily orthonormal (off-axis frusta are expressible).
 * Output pixel (i,j) of a W x H view looks along
 *   D = fwd + ((2(i+.5)/W - 1) tan_half_x) right + ((2(j+.5)/H - 1) tan_half_y) down
 * from eye, in the light slab's world frame (camera plane z = 0, image plane z = z_st). */
typedef struct {
    float eye[3], right[3], down[3], fwd[3];
    float tan_half_x, tan_half_y;
    float _pad[2];
} hmlfc_camera; /* 64 bytes */

/* Algorithmic-bytes accounting of one render or decode batch: every distinct
 * (plane-channel, block) touched -- including reference blocks reached through motion
 * vectors -- counts once. */
typedef struct {
    int64_t blocks_touched;
    int64_t flag_bits;       /* 1 bit per touched block of a reference plane, 2 of a predictive one */
    int64_t payload_bits15;  /* payload bits of touched significant blocks, in units of 1/15 bit    */
    int64_t mv_bits15;       /* motion-record bits of touched predicted blocks, in 1/15 bit         */
    int64_t rkv_bytes;       /* distinct top-level RKV samples touched: 1 (Y) or 2 (Co,Cg) bytes    */
    int64_t out_bytes, in_bytes;
    double bytes_alg;        /* total bytes                                                          */
} hmlfc_footprint_t;

/* hmlfc_load -- PAPER.md:293 "the top-level RKV images are decoded and stored in memory",
 * PAPER.md:296 "the reference SRV images at all the levels are ... loaded into the memory".
 * Parses the serialized stream (layout: DESIGN.md "Stream format v1"), re-packs it into the
 * device structure-of-arrays form (flag + rank records, bit-packed BISE payloads and motion
 * vectors, packed top-level RKVs) and uploads it to the current CUDA device.  For streams with
 * full-resolution chroma one kernel then writes the BLOCK RECORDS on the device (every stored value
 * and motion record once more, grouped per block for random access: DESIGN.md section 8); the call
 * returns when they are complete.  Streams with subsampled chroma (header byte 49, R18) and with half-pel
 * motion offsets (byte 55, R28) get no block records, but every entry point has an instantiation of a fast kernel for
 * them: hmlfc_decode the warp-cooperative kernel on the stream's strings (any block size), hmlfc_render and hmlfc_decode_views / _blocks
 * the tile and block-row kernels for 4 x 4 blocks (hmlfc_render: not both flags at once, half-pel windows up to 63); other cases run
 * per sample -- identical bytes.  hmlfc_info().device_bytes counts everything that stays resident
 * (about 2.2 x the stream).  HMLFC_E_NOMEM if the device cannot hold it.
 *   h_stream_bytes : host, read only during the call; the caller may free it afterwards.
 *   out            : receives the handle; untouched on error.                              */
int hmlfc_load(const void *h_stream_bytes, size_t len, hmlfc_handle **out);

int hmlfc_info(const hmlfc_handle *h, hmlfc_info_t *out);

/* hmlfc_decode -- PAPER.md:289-293 (decoding procedure) and :309 (random access): for each
 * coordinate, top-level RKV sample + sum over the levels of the SRV sample (stored block value,
 * plus or minus the motion-shifted reference-SRV sample for predicted blocks), inverse YCoCg-R,
 * clamp to [0,255].
 *   d_coords : device, int32 [n][4] = (u, v, s, t), row-major.
 *   d_out    : device, uint8 [n][3] RGB.
 * An out-of-range coordinate writes (0,0,0) and increments the handle's out-of-range counter. */
int hmlfc_decode(const hmlfc_handle *h, const int32_t *d_coords, int64_t n, uint8_t *d_out, void *cuda_stream);

/* hmlfc_decode_views -- the same decoding procedure for WHOLE views: every pixel of view (u, v) = d_views[k], in
 * row-major order ("parallel decompression of different pixel values"; the dense counterpart of hmlfc_decode: no
 * 16-byte coordinate per sample is read, neighbouring lanes decode neighbouring pixels).
 *   d_views : device, int32 [n_views][2] = (u, v).
 *   d_out   : device, uint8 [n_views][Ht][Ws][3] RGB.
 * A view outside the camera grid is written black and every pixel of it counted as out of range.  Progressive decoding
 * (hmlfc_set_min_level) applies.  Asynchronous like hmlfc_decode.  B = 4 streams run one lane per block-row segment (4 pixels);
 * other block sizes, and any stream after hmlfc_set_decode_variant(h, 1 or 2), one lane per pixel -- identical bytes. */
int hmlfc_decode_views(const hmlfc_handle *h, const int32_t *d_views, int64_t n_views, uint8_t *d_out, void *cuda_stream);

/* hmlfc_decode_blocks -- random access at the granularity the paper decodes at ("As a block of pixels are decoded, our
 * method benefits any LF rendering scheme by providing fast access to neighboring pixels"): whole B x B blocks.
 *   d_blocks : device, int32 [n][4] = (u, v, bx, by): block column / row inside view (u, v), 0 <= bx < Ws/B, 0 <= by < Ht/B.
 *   d_out    : device, uint8 [n][B][B][3] RGB (row-major inside the block).
 * A block outside the light field is written black and its B^2 pixels counted as out of range.  Progressive decoding applies.
 * Asynchronous like hmlfc_decode; B = 4 streams run one lane per block row, others one lane per pixel -- identical bytes. */
int hmlfc_decode_blocks(const hmlfc_handle *h, const int32_t *d_blocks, int64_t n_blocks, uint8_t *d_out, void *cuda_stream);

/* hmlfc_render -- PAPER.md:73 / :309 / :409: per output pixel, ray -> (u,v,s,t) on the two
 * planes, 16-tap quadrilinear blend of decoded samples (4 nearest views x 4 nearest pixels,
 * edge-clamped), rounded to RGB8; rays that miss the slab get the background colour.
 *   d_cameras : device, hmlfc_camera [n_views].
 *   d_out     : device, uint8 [n_views][H][W][3], row-major, no padding.                    */
int hmlfc_render(const hmlfc_handle *h, const hmlfc_camera *d_cameras, int n_views, int W, int H, uint8_t *d_out,
                 void *cuda_stream);

/* hmlfc_render_noalloc -- hmlfc_render for callers that cannot allocate (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): the same views, byte for byte, from the tile kernels (tile_tables_kernel + render_tiles_kernel)
 * with the tile tables -- the scratch memory hmlfc_render takes from a stream-ordered pool -- in a static device buffer of the library.
 * The call launches two kernels on cuda_stream and calls no cudaMalloc, cudaFree or other allocating routine.
 *   Limit: n_views x ceil(W / w) x ceil(H / 32) <= HMLFC_NOALLOC_MAX_TILES tiles per call (w = 64 where W x H >= 8 x Ws x Ht on streams
 *   with full-resolution chroma and whole-pixel motion, else 32),
 *   e.g. 16 views of 512 x 512; beyond it HMLFC_E_LIMIT and nothing is launched -- render the views in several calls.  The buffer
 *   (HMLFC_NOALLOC_MAX_TILES x 3,200 bytes = 13.1 MB) is held by every GPU that loads the library until the process exits.
 *   Streams: 4 x 4 blocks (the streams whose hmlfc_render uses scratch memory at all), chroma-subsampled or half-pel ones included
 *   (not both at once; half-pel windows up to 63); others HMLFC_E_UNSUPPORTED.  The current device must be the handle's (hmlfc_load sets the buffer up for its device).
 *   All calls on a device share the buffer: calls that may OVERLAP on the GPU (different streams without a dependency) race on it
 *   and give undefined pixels; calls on one stream, or ordered by events, are safe.  Progressive decoding applies. */
#define HMLFC_NOALLOC_MAX_TILES 4096
int hmlfc_render_noalloc(const hmlfc_handle *h, const hmlfc_camera *d_cameras, int n_views, int W, int H, uint8_t *d_out,
                         void *cuda_stream);

/* hmlfc_render_lod -- level of detail per view ("progressive decoding"; R26, R27): view k is rendered as by
 * hmlfc_render with the tree walk stopped above level max(h_levels[k], the handle's min_level), i.e. from the representative key views of
 * its level-h_levels[k] clusters: fewer lookups and bytes per sample for views that need less angular detail.
 *   h_levels : HOST, int32 [n_views], each in [0, height]; the other arguments as for hmlfc_render.
 * One kernel sequence per run of consecutive views with equal level, on `cuda_stream`; asynchronous.  HMLFC_E_INVALID for a level
 * outside [0, height].
 * hmlfc_lod_levels -- the distance rule that fills such an array (host arithmetic only): a viewer at distance d = |z_st - eye.z| from the
 * image plane gets floor(log2(d / d0)) clamped to [0, height] (every doubling of the distance beyond d0 goes one level up); d0 <= 0
 * gives level 0 everywhere.   h_cameras : HOST, hmlfc_camera [n_views];  h_levels : HOST, int32 [n_views] (out). */
int hmlfc_render_lod(const hmlfc_handle *h, const hmlfc_camera *d_cameras, const int32_t *h_levels, int n_views, int W, int H,
                     uint8_t *d_out, void *cuda_stream);
int hmlfc_lod_levels(const hmlfc_handle *h, const hmlfc_camera *h_cameras, int n_views, float d0, int32_t *h_levels);

/* End-to-end variants with HOST buffers: copy the inputs to the device, run the same kernels,
 * copy the result back, synchronise.  Scratch device buffers live in the handle and grow on
 * demand (so these calls are not re-entrant on one handle).  The work is pipelined in
 * chunks (whole views / >= 2^20 coordinates) over three streams of the handle, so the input
 * copy of one chunk, the kernel of the previous and the result copy of the one before overlap
 * (hmlfc_render_host alternates its chunks' kernels between two streams so that their last waves overlap);
 * the bytes written equal those of one whole-batch call.  Pinned host memory makes the copies
 * asynchronous DMA; pageable memory works too (the copies then serialise). */
int hmlfc_decode_host(hmlfc_handle *h, const int32_t *h_coords, int64_t n, uint8_t *h_out);
int hmlfc_decode_views_host(hmlfc_handle *h, const int32_t *h_views, int64_t n_views, uint8_t *h_out);
int hmlfc_render_host(hmlfc_handle *h, const hmlfc_camera *h_cameras, int n_views, int W, int H, uint8_t *h_out);

/* Synchronous: the number of out-of-range coordinates seen by hmlfc_decode since load. */
int hmlfc_last_oob_count(const hmlfc_handle *h, int64_t *out);

/* Measurement aid (not on the hot path): marks every block / RKV sample the batch touches with
 * a kernel, then reduces the marks to the algorithmic-byte count.  Synchronous. */
int hmlfc_footprint_render(hmlfc_handle *h, const hmlfc_camera *d_cameras, int n_views, int W, int H,
                           hmlfc_footprint_t *out);
int hmlfc_footprint_decode(hmlfc_handle *h, const int32_t *d_coords, int64_t n, hmlfc_footprint_t *out);

/* Kernel selection for hmlfc_render (A/B measurements and cross-checks; all variants produce identical
 * bytes): 0 = automatic (default; for B = 4 streams 11, 12 or 7 as described below, else 4), 1 = one thread per
 * output pixel (16 independent tap decodes -- the unshared definition, kept as the cross-check), 4 / 5 = a
 * block-centric pipeline run by ONE WARP per 16 x 8 / 8 x 8 tile.  The two fused kernels for 4 x 4 blocks
 * (per-view footprint boxes, block-ROW tasks: 4 BISE values per lane from two 64-bit windows):
 * 6 .. 10 = the general kernel (tile tables built inside the CTA, quadtree of sub-tile passes): 256 threads per
 * 32 x 32 tile with a 65 KB (3 CTAs per SM) / 103 KB (2) / 46 KB (4) shared-memory arena, 1024 threads per
 * 64 x 64 tile, 512 threads per 64 x 32 tile; 11 .. 15 = the tile kernel (tables of all tiles from a kernel of
 * their own, one pass per tile; two launches per call and a scratch buffer from the library's stream-ordered
 * pool): 32 x 32 tile with 3 / 4 CTAs per SM, 64 x 32 tile with 512 threads, 64 x 32 tile with 256 threads (8
 * pixels per thread) and 2 / 3 CTAs per SM.  The automatic choice takes 7 when a view has fewer than twice the
 * pixels of a light-field image (little magnification: many samples per tile), 15 when it has at least eight
 * times as many, else 11.  On streams with subsampled chroma or half-pel motion offsets (4 x 4 blocks) 0 and 6 .. 15 all run the
 * tile kernel's instantiation for that kind of stream (32 x 32 tiles, 3 CTAs per SM); 4 / 5 and other block sizes run per pixel. */
int hmlfc_set_render_variant(hmlfc_handle *h, int variant);

/* Progressive decoding (PAPER.md:57, :183 name the property; R26): hmlfc_decode / hmlfc_render sum the top-level RKV and the
 * levels height-1 .. min_level only -- the walk from the root stops early.  0 (default) = full quality; `height` = the top-level RKV
 * alone; level L yields the representative key view of the level-L cluster containing the view.  Fewer levels = fewer lookups and
 * bytes per sample.  Takes effect for launches enqueued afterwards; HMLFC_E_INVALID outside [0, height]. */
int hmlfc_set_min_level(hmlfc_handle *h, int min_level);

/* Kernel selection for hmlfc_decode (identical bytes): 0 = automatic (default), 1 = one thread per
 * coordinate walks the tree on its own, 2 / 3 / 4 = warp-cooperative (each lane classifies its coordinate, the
 * motion-record and value decodes run as 32-wide batches from per-warp task stacks): 2 reads the three
 * channels' flag records and descriptors of every level up front, 3 reads ONE 32-byte sector of flag words per
 * level and lets the tasks of significant blocks fetch the rest; 4 reads the BLOCK RECORDS hmlfc_load builds for
 * streams with full-resolution chroma and whole-pixel motion (every stored value and motion record once more, as plain binary fields
 * grouped per block: one sector per level says what a plane holds for a sample and where, one or two more hold
 * all three channels of it; counted in device_bytes).  The automatic choice is 4 where the stream has block
 * records; chroma-subsampled and half-pel streams have none and run, for 0 and 2 .. 4 alike, the instantiation of kernel 2 for that kind of
 * stream; otherwise 3 for streams whose device form fits the L2 cache and where at most a quarter of the block flags are set, else 2.
 * hmlfc_decode_views / _blocks: 0 = the block-row kernel (4 x 4 blocks), anything else their lane-per-pixel kernels. */
int hmlfc_set_decode_variant(hmlfc_handle *h, int variant);

/* Encoder side (first "next" row): phase-shifted exhaustive block motion search, PAPER.md:227-248,
 * Eqs. (1)-(2).  For pair k = (p, r) = d_pairs[k] and every block x block block of plane p, over all motion vectors
 * (dx, dy) in [-window, window]^2:
 *     Delta-(dx,dy) = sum |P(x,y) - R(x+dx, y+dy)|,   Delta+(dx,dy) = sum |P(x,y) + R(x+dx, y+dy)|,
 * R reading 0 outside the image; the result is the minimum over both modes, ties resolved subtractive before additive
 * ("phase-shifted"), then smallest dy, then smallest dx (R8, R9).
 *   d_planes  device, int16 [n_planes][Ht][Ws] (SRV images of one level and channel, any order)
 *   d_pairs   device, int32 [n_pairs][2] = (index of the predictive plane, index of its reference plane)
 *   d_out     device, int32 [n_pairs][Ht/block][Ws/block][4] = mode (0 subtractive, 1 additive), dx, dy, Delta
 * Needs no handle (the encoder has no stream yet).  Enqueues on cuda_stream and returns; block in 1..8 must divide
 * Ws and Ht, window <= 64, n_pairs <= 65535, else HMLFC_E_UNSUPPORTED.  Integer-exact for any int16 input. */
int hmlfc_search(const int16_t *d_planes, const int32_t *d_pairs, int n_pairs, int Ws, int Ht, int block, int window,
                 int32_t *d_out, void *cuda_stream);

/* Encoder side, hierarchy build (SURVEY.md 8(f) rank 1 with hmlfc_search): forward YCoCg-R and the RLFC
 * hierarchy of PAPER.md:200 (section 4.3): 2 x 2 clusters on the camera grid, RKV = uniform mean of the members present
 * rounded half away from zero, SRV = member - RKV, repeated `height` times.  Level L has U_L x V_L planes,
 * U_L = ceil(U / 2^L); plane (pu, pv) of a level has index pv * U_L + pu.
 *   d_lf   device, uint8 [V][U][Ht][Ws][3] RGB8 (4-byte aligned)
 *   d_srv  device, int16 [3][n_srv_planes][Ht][Ws]: channel (Y, Co, Cg) outermost, then the SRV planes of level 0, level 1, ..
 *          level height-1 (n_srv_planes = sum_{L<height} U_L V_L)
 *   d_x    device, int16 [3][n_x_planes][Ht][Ws]: the RKV planes X_1 .. X_height (n_x_planes = sum_{1<=L<=height} U_L V_L);
 *          the last U_h V_h planes of each channel are the top-level RKVs
 * hmlfc_hierarchy_sizes (host only) returns the two plane counts.  hmlfc_hierarchy enqueues `height` kernels on cuda_stream and
 * returns; Ws must be a multiple of 4 (HMLFC_E_UNSUPPORTED), the outputs 8-byte aligned.  Integer-exact. */
int hmlfc_hierarchy_sizes(int U, int V, int height, int64_t *n_srv_planes, int64_t *n_x_planes);
int hmlfc_hierarchy(const uint8_t *d_lf, int U, int V, int Ws, int Ht, int height, int16_t *d_srv, int16_t *d_x, void *cuda_stream);

/* Encoder, complete: RGB8 light field on the device -> compressed stream in host memory, every
 * arithmetic step in CUDA kernels: hmlfc_hierarchy, hmlfc_search for every predictive SRV image of every
 * level and channel, the replacement step and the two block thresholds (reference block
 * kept iff sum|block| >= tau_ref; predictive block per `policy`, R13: 0 adaptive, 1 all, 2 literal, 3 no motion
 * compensation at all = the RLFC hierarchy alone), BISE packing of
 * the stored blocks and of the joint motion records, in the BFS order of PAPER.md:276.  The host writes the
 * header, the raw top-level RKVs and the directory around the device-built sections ("Stream format v1").
 *   d_lf      device, uint8 [V][U][Ht][Ws][3] RGB8, 4-byte aligned (not modified)
 *   p         host; block in {2,4,8} dividing Ws and Ht, Ws % 4 == 0, height <= 8, window <= 64 (else HMLFC_E_UNSUPPORTED);
 *             geometry / background / seed are copied into the header
 *   h_stream  receives a malloc'ed buffer of *len bytes that hmlfc_load accepts; release it with hmlfc_stream_free
 *   stats     optional (may be NULL): device time per phase (CUDA events) and block counts
 * Synchronous (the value ranges must reach the host before the strings can be laid out); its device scratch (about 2.7 x the
 * raw light field as int16 planes + 16 bytes per predictive block) comes from a stream-ordered pool (see
 * hmlfc_encode_release_scratch). */
typedef struct {
    int32_t U, V, Ws, Ht, height, block, window, tau_ref, tau_res, policy;
    float uv_origin[2], uv_step[2], st_origin[2], st_step[2], z_st;
    unsigned char background[3], _pad;
    uint64_t seed;
} hmlfc_encode_params_t;
typedef struct {
    float ms_hierarchy, ms_search, ms_classify, ms_pack;   /* device time of the four phases */
    float ms_wall, ms_assemble;                            /* host wall clock: the whole call; stream assembly + copies to the host */
    int64_t n_plane_channels, n_res_blocks, n_pred_blocks, n_search_blocks;
    int32_t kernel_launches, cuda_error;
    int64_t sse;                  /* sum of squared RGB differences between the stream's reconstruction and the input */
    double psnr;                  /* 10 log10(255^2 / (sse / bytes)); +inf when sse = 0 */
    int32_t tau_ref, tau_res;     /* the thresholds written to the stream */
    int32_t bisection_steps, _pad;
} hmlfc_encode_stats_t;
int hmlfc_encode(const uint8_t *d_lf, const hmlfc_encode_params_t *p, uint8_t **h_stream, size_t *len,
                 hmlfc_encode_stats_t *stats, void *cuda_stream);
/* The same with the thresholds chosen for a quality target ("encoding parameters are varied ... to achieve a
 * similar compression quality"; W3, R24): bisection of tau_res over [0, 4096] with tau_ref = floor(tau_res / 2), at most
 * max_iter steps, until the PSNR of the reconstruction (what hmlfc_decode returns for the stream, computed by a kernel from the
 * encoder's planes) is within tol dB of target_psnr; the closest step wins.  p's tau_ref / tau_res are ignored.  Hierarchy and
 * search run once.  HMLFC_E_INVALID for a negative or non-finite target, tol < 0 or max_iter < 1. */
int hmlfc_encode_psnr(const uint8_t *d_lf, const hmlfc_encode_params_t *p, double target_psnr, double tol, int max_iter,
                      uint8_t **h_stream, size_t *len, hmlfc_encode_stats_t *stats, void *cuda_stream);
void hmlfc_stream_free(uint8_t *h_stream);
/* hmlfc_encode keeps its device scratch in a stream-ordered memory pool of the current device between calls (a second call
 * allocates nothing from the driver); this returns it.  Synchronises the device. */
int hmlfc_encode_release_scratch(void);

/* Number of kernels this library has launched through the handle since load (bench accounting). */
int hmlfc_launch_count(const hmlfc_handle *h, int64_t *out);

void hmlfc_free(hmlfc_handle *h);
const char *hmlfc_strerror(int code);
/* cudaError_t of the most recent failed CUDA call made through this handle (0 if none). */
int hmlfc_last_cuda_error(const hmlfc_handle *h);

#ifdef __cplusplus
}
#endif
#endif /* HMLFC_H */
