// C ABI of libhmlfc_b200.so (include/hmlfc.h): stream parsing, device upload, kernel dispatch.
// The stream byte layout parsed here is DESIGN.md "Stream format v1"; this parser is written
// from that document and shares no code with the oracle's.
#include "../../include/hmlfc.h"
#include "hmlfc_kernels.cuh"
#include "hmlfc_tables.h"

#include <atomic>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

using namespace hmlfc;

struct hmlfc_handle {
    DevStream ds{};
    hmlfc_info_t info{};
    int device = 0;
    // device allocations
    uint4 *d_pc = nullptr;
    uint4 *d_flagrec = nullptr;
    uint4 *d_bslot = nullptr;
    uint4 *d_pb = nullptr;              // block records (hmlfc_device.cuh): per-plane descriptors and the records
    uint32_t *d_brec = nullptr;
    uint32_t *d_pay = nullptr;
    uint32_t *d_mv = nullptr;
    short4 *d_rkv = nullptr;
    uint32_t *d_bits15 = nullptr;       // per plane-channel BISE bits/value in 1/15 bit (footprint only)
    unsigned long long *d_oob = nullptr;
    uint64_t n_pc = 0;
    uint32_t mv_bits15 = 0;
    // scratch of the *_host entry points
    void *d_in = nullptr;
    size_t d_in_cap = 0;
    uint8_t *d_outbuf = nullptr;
    size_t d_out_cap = 0;
    cudaStream_t host_stream = nullptr;   // kernels of the *_host entry points
    cudaStream_t in_stream = nullptr;     // host -> device copies (own copy engine)
    cudaStream_t out_stream = nullptr;    // device -> host copies (own copy engine)
    static constexpr int kMaxChunks = 32;
    cudaEvent_t ev_in[kMaxChunks] = {};   // chunk c's input is on the device
    cudaEvent_t ev_done[kMaxChunks] = {}; // chunk c's kernel has finished
    int render_variant = 0;
    int decode_variant = 0;
    mutable std::atomic<long long> launches{0};
    mutable std::atomic<int> last_cuda_error{0};
};

namespace hmlfc {

static cudaMemPool_t g_pool[64] = {};

cudaError_t scratch_pool(cudaMemPool_t *out)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    if (!g_pool[dev]) {
        cudaMemPoolProps props{};
        props.allocType = cudaMemAllocationTypePinned;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        if ((e = cudaMemPoolCreate(&g_pool[dev], &props)) != cudaSuccess) return e;
        uint64_t keep = ~0ull;  // keep freed scratch for the next call (hmlfc_encode_release_scratch returns it)
        if ((e = cudaMemPoolSetAttribute(g_pool[dev], cudaMemPoolAttrReleaseThreshold, &keep)) != cudaSuccess) return e;
    }
    *out = g_pool[dev];
    return cudaSuccess;
}

cudaError_t scratch_pool_trim()
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    if (!g_pool[dev]) return cudaSuccess;
    if ((e = cudaDeviceSynchronize()) != cudaSuccess) return e;
    return cudaMemPoolTrimTo(g_pool[dev], 0);
}

}  // namespace hmlfc

namespace {

int cuda_fail(const hmlfc_handle *h, cudaError_t e)
{
    if (h) h->last_cuda_error.store((int)e);
    return HMLFC_E_CUDA;
}

#define CU(h, call)                                            \
    do {                                                       \
        cudaError_t e__ = (call);                              \
        if (e__ != cudaSuccess) return cuda_fail((h), e__);    \
    } while (0)

void release(hmlfc_handle *h)
{
    if (!h) return;
    cudaFree(h->d_pc); cudaFree(h->d_flagrec); cudaFree(h->d_pb); cudaFree(h->d_bslot); cudaFree(h->d_brec); cudaFree(h->d_pay); cudaFree(h->d_mv); cudaFree(h->d_rkv);
    cudaFree(h->d_bits15); cudaFree(h->d_oob); cudaFree(h->d_in); cudaFree(h->d_outbuf);
    if (h->host_stream) cudaStreamDestroy(h->host_stream);
    if (h->in_stream) cudaStreamDestroy(h->in_stream);
    if (h->out_stream) cudaStreamDestroy(h->out_stream);
    for (int i = 0; i < hmlfc_handle::kMaxChunks; ++i) {
        if (h->ev_in[i]) cudaEventDestroy(h->ev_in[i]);
        if (h->ev_done[i]) cudaEventDestroy(h->ev_done[i]);
    }
    delete h;
}

cudaError_t create_events(hmlfc_handle *h)
{
    for (int i = 0; i < hmlfc_handle::kMaxChunks; ++i) {
        cudaError_t e;
        if ((e = cudaEventCreateWithFlags(&h->ev_in[i], cudaEventDisableTiming)) != cudaSuccess) return e;
        if ((e = cudaEventCreateWithFlags(&h->ev_done[i], cudaEventDisableTiming)) != cudaSuccess) return e;
    }
    return cudaSuccess;
}

template <typename T>
cudaError_t upload(T **dst, const void *src, size_t bytes, size_t slack, uint64_t *total)
{
    cudaError_t e = cudaMalloc(reinterpret_cast<void **>(dst), bytes + slack);
    if (e != cudaSuccess) return e;
    if (slack && (e = cudaMemset(reinterpret_cast<uint8_t *>(*dst) + bytes, 0, slack)) != cudaSuccess) return e;
    if (bytes && (e = cudaMemcpy(*dst, src, bytes, cudaMemcpyHostToDevice)) != cudaSuccess) return e;
    *total += bytes + slack;
    return cudaSuccess;
}

}  // namespace

extern "C" {

const char *hmlfc_strerror(int code)
{
    switch (code) {
    case HMLFC_OK: return "ok";
    case HMLFC_E_MAGIC: return "bad magic: not an HMLF stream";
    case HMLFC_E_TRUNCATED: return "truncated stream";
    case HMLFC_E_VERSION: return "unsupported stream version";
    case HMLFC_E_INVALID: return "invalid argument";
    case HMLFC_E_UNSUPPORTED: return "unsupported stream parameter";
    case HMLFC_E_CORRUPT: return "corrupt stream directory";
    case HMLFC_E_NOMEM: return "out of memory";
    case HMLFC_E_CUDA: return "CUDA runtime error";
    case HMLFC_E_LIMIT: return "request exceeds a fixed capacity of this entry point";
    default: return "unknown error";
    }
}

int hmlfc_load(const void *h_stream_bytes, size_t len, hmlfc_handle **out)
{
    if (!h_stream_bytes || !out) return HMLFC_E_INVALID;
    HostTables T;
    int rc = build_tables(h_stream_bytes, len, T);
    if (rc != HMLFC_OK) return rc;
    hmlfc_handle *h = new (std::nothrow) hmlfc_handle();
    if (!h) return HMLFC_E_NOMEM;
    h->ds = T.ds;
    h->info = T.info;
    h->n_pc = T.n_pc;
    h->mv_bits15 = T.mv_bits15;
    const uint8_t *s = static_cast<const uint8_t *>(h_stream_bytes);

    cudaError_t ce;
    uint64_t dev_bytes = 0;
    if ((ce = cudaGetDevice(&h->device)) != cudaSuccess ||
        (ce = upload(&h->d_pc, T.pc.data(), T.pc.size() * sizeof(uint4), 0, &dev_bytes)) != cudaSuccess ||
        (ce = upload(&h->d_flagrec, T.flagrec.data(), T.flagrec.size() * sizeof(uint4), 0, &dev_bytes)) != cudaSuccess ||
        (ce = upload(&h->d_pay, s + T.off_pay, (size_t)(T.off_mv - T.off_pay), 64, &dev_bytes)) != cudaSuccess ||
        (ce = upload(&h->d_mv, s + T.off_mv, (size_t)(T.total - T.off_mv), 64, &dev_bytes)) != cudaSuccess ||
        (ce = upload(&h->d_rkv, T.rkv.data(), T.rkv.size() * sizeof(short4), 0, &dev_bytes)) != cudaSuccess ||
        (ce = upload(&h->d_bits15, T.bits15.data(), T.bits15.size() * sizeof(uint32_t), 0, &dev_bytes)) != cudaSuccess ||
        (ce = cudaMalloc(reinterpret_cast<void **>(&h->d_oob), sizeof(unsigned long long))) != cudaSuccess ||
        (ce = cudaMemset(h->d_oob, 0, sizeof(unsigned long long))) != cudaSuccess ||
        (ce = cudaStreamCreateWithFlags(&h->host_stream, cudaStreamNonBlocking)) != cudaSuccess ||
        (ce = cudaStreamCreateWithFlags(&h->in_stream, cudaStreamNonBlocking)) != cudaSuccess ||
        (ce = cudaStreamCreateWithFlags(&h->out_stream, cudaStreamNonBlocking)) != cudaSuccess ||
        (ce = create_events(h)) != cudaSuccess ||
        (ce = configure_render_warp()) != cudaSuccess || (ce = configure_render_cta()) != cudaSuccess ||
        (ce = configure_render_tiles()) != cudaSuccess || (ce = configure_decode_queue()) != cudaSuccess ||
        (ce = configure_render_tiles_noalloc()) != cudaSuccess) {
        const int code = (ce == cudaErrorMemoryAllocation) ? HMLFC_E_NOMEM : HMLFC_E_CUDA;
        release(h);
        return code;
    }
    DevStream &D = h->ds;
    D.pc = h->d_pc; D.flagrec = h->d_flagrec; D.pay = h->d_pay; D.mv = h->d_mv; D.rkv = h->d_rkv;
    D.pb = nullptr; D.bslot = nullptr; D.brec = nullptr;
    if (!T.pb.empty()) {
        // block records: every stored value and motion record once more, regrouped per block (one kernel over the uploaded stream)
        const size_t bytes = (size_t)T.brec_words * 4;
        if ((ce = upload(&h->d_pb, T.pb.data(), T.pb.size() * sizeof(uint4), 0, &dev_bytes)) != cudaSuccess ||
            (ce = upload(&h->d_bslot, T.bslot.data(), T.bslot.size() * sizeof(uint4), 0, &dev_bytes)) != cudaSuccess ||
            (ce = cudaMalloc(reinterpret_cast<void **>(&h->d_brec), bytes)) != cudaSuccess ||
            (ce = cudaMemsetAsync(h->d_brec, 0, bytes, h->host_stream)) != cudaSuccess) {
            const int code = (ce == cudaErrorMemoryAllocation) ? HMLFC_E_NOMEM : HMLFC_E_CUDA;
            release(h);
            return code;
        }
        D.pb = h->d_pb; D.bslot = h->d_bslot;
        if ((ce = launch_repack(D, T.pb.size(), h->d_brec, h->host_stream)) != cudaSuccess ||
            (ce = cudaStreamSynchronize(h->host_stream)) != cudaSuccess) {
            release(h);
            return HMLFC_E_CUDA;
        }
        D.brec = h->d_brec;
        dev_bytes += bytes;
    }
    h->info.device_bytes = dev_bytes;
    // hmlfc_decode's classification: one flag sector per level and everything else fetched by the tasks pays where the L2 holds the stream
    // (126 MB on B200; coordinates and output pass through it too) and few blocks carry data (measured: cfg2, 17% of the flags set,
    // 12.7 -> 14.4 G px/s; cfg3, denser, 8.4 -> 7.3; cfg4 / cfg5 in HBM 6.4 -> 5.2 / 4.0 -> 3.3)
    D.l2_resident = (dev_bytes <= (96ull << 20) && 4 * T.n_flagged <= T.n_pc * (uint64_t)D.nblk) ? 1u : 0u;
    *out = h;
    return HMLFC_OK;
}

int hmlfc_info(const hmlfc_handle *h, hmlfc_info_t *out)
{
    if (!h || !out) return HMLFC_E_INVALID;
    *out = h->info;
    return HMLFC_OK;
}

int hmlfc_decode(const hmlfc_handle *h, const int32_t *d_coords, int64_t n, uint8_t *d_out, void *cuda_stream)
{
    if (!h || n < 0 || (n > 0 && (!d_coords || !d_out))) return HMLFC_E_INVALID;
    int nl = 0;
    if (h->decode_variant == 1)  // the per-sample kernel (cross-check)
        CU(h, launch_decode(h->ds, d_coords, n, d_out, h->d_oob, static_cast<cudaStream_t>(cuda_stream), &nl));
    else
        CU(h, launch_decode_queue(h->ds, d_coords, n, d_out, h->d_oob, static_cast<cudaStream_t>(cuda_stream), &nl,
                                  h->decode_variant == 2 ? 0 : h->decode_variant == 3 ? 1 : h->decode_variant == 4 ? 2 : -1));
    h->launches += nl;
    return HMLFC_OK;
}

int hmlfc_decode_views(const hmlfc_handle *h, const int32_t *d_views, int64_t n_views, uint8_t *d_out, void *cuda_stream)
{
    if (!h || n_views < 0 || (n_views > 0 && (!d_views || !d_out))) return HMLFC_E_INVALID;
    int nl = 0;
    // B = 4 streams: one lane per block-row segment; other block sizes (and decode variant 1 / 2, for cross-checks): one lane per pixel
    // (half-pel and chroma-subsampled streams, R28 / R18: the block-row kernel's instantiations; per sample for other block sizes and as a cross-check)
    if ((h->ds.cs || h->ds.sp) && !(h->ds.B == 4 && h->decode_variant == 0))
        CU(h, launch_decode_dense(h->ds, d_views, n_views, false, d_out, h->d_oob, static_cast<cudaStream_t>(cuda_stream), &nl));
    else if (h->ds.B == 4 && h->decode_variant == 0)
        CU(h, launch_decode_rows(h->ds, d_views, n_views, d_out, h->d_oob, static_cast<cudaStream_t>(cuda_stream), &nl));
    else
        CU(h, launch_decode_views(h->ds, d_views, n_views, d_out, h->d_oob, static_cast<cudaStream_t>(cuda_stream), &nl));
    h->launches += nl;
    return HMLFC_OK;
}

int hmlfc_decode_blocks(const hmlfc_handle *h, const int32_t *d_blocks, int64_t n_blocks, uint8_t *d_out, void *cuda_stream)
{
    if (!h || n_blocks < 0 || (n_blocks > 0 && (!d_blocks || !d_out))) return HMLFC_E_INVALID;
    int nl = 0;
    if ((h->ds.cs || h->ds.sp) && !(h->ds.B == 4 && h->decode_variant == 0))
        CU(h, launch_decode_dense(h->ds, d_blocks, n_blocks, true, d_out, h->d_oob, static_cast<cudaStream_t>(cuda_stream), &nl));
    else if (h->ds.B == 4 && h->decode_variant == 0)
        CU(h, launch_decode_block_rows(h->ds, d_blocks, n_blocks, d_out, h->d_oob, static_cast<cudaStream_t>(cuda_stream), &nl));
    else
        CU(h, launch_decode_blocks(h->ds, d_blocks, n_blocks, d_out, h->d_oob, static_cast<cudaStream_t>(cuda_stream), &nl));
    h->launches += nl;
    return HMLFC_OK;
}

// hmlfc_render with the stream view D (= D, or D with another lmin: per-view level of detail)
static int render_impl(const hmlfc_handle *h, const DevStream &D, const hmlfc_camera *d_cameras, int n_views, int W, int H, uint8_t *d_out,
                       void *cuda_stream)
{
    if (!h || n_views < 0 || W <= 0 || H <= 0 || n_views > 65535 || (n_views > 0 && (!d_cameras || !d_out))) return HMLFC_E_INVALID;
    static_assert(sizeof(hmlfc_camera) == sizeof(Camera) && sizeof(Camera) == 64, "camera layout");
    int nl = 0;
    const Camera *cams = reinterpret_cast<const Camera *>(d_cameras);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    // progressive decoding (lmin > 0) is implemented by the thread-per-pixel kernel and the two fused kernels for 4 x 4 blocks
    const int rv = h->render_variant;
    const bool fused_ok = D.B == 4 && (rv == 0 || (rv >= 6 && rv <= 15));
    // half-pel streams (R28): the tile kernel's half-pel instantiation (32 x 32 tiles) for 4 x 4 blocks and windows up to 63, else per sample
    const bool sp_tiles = D.sp && !D.cs && D.B == 4 && D.mv_off <= 127 && (rv == 0 || rv >= 6);
    // chroma-subsampled streams (R18): likewise its chroma instantiation (not both at once)
    const bool cs_tiles = D.cs && !D.sp && D.B == 4 && (rv == 0 || rv >= 6);
    if (rv == 1 || (D.cs && !cs_tiles) || (D.sp && !sp_tiles) || (D.lmin > 0 && !fused_ok))
        CU(h, launch_render_pixel(D, cams, n_views, W, H, d_out, st, &nl));
    else if (rv == 4 || rv == 5 || D.B != 4)
        CU(h, launch_render_warp(D, cams, n_views, W, H, d_out, st, &nl, rv == 5 ? 1 : 0));
    else {
        // 0: chosen from the sizes -- views that look at about as many light-field samples as they have pixels (or more) go to the general
        // kernel with its largest arena, the others to the tile kernel (tables from a kernel of their own); 6 .. 10: the general kernel's five
        // configurations; 11 / 12: the tile kernel with 3 / 4 CTAs per SM.  All give identical bytes.
        int tiles = rv >= 11 && rv <= 15 ? rv - 11 : -1;
        // measured, ms per step (tile kernel 32 x 32 x 3 CTAs / 32 x 32 x 4 CTAs / 64 x 32 with 512 threads / 64 x 32 with 256 threads x 2 CTAs /
        // 64 x 32 with 256 threads x 3 CTAs, against the general kernel's best configuration): cfg2 0.66 / 0.93 / 0.67 / 0.70 / 1.09 (0.81),
        // cfg4 0.88 / 1.26 / 0.90 / 0.97 / 1.39 (1.00), cfg5 1.18 / 1.07 / 1.05 / 1.18 / 0.97 (1.50); cfg3 (about one sample per pixel) 1.06 / 1.28 /
        // 1.12 / 1.44 / 1.50 (0.84)
        if (rv == 0 && (long long)W * H >= 2LL * D.Ws * D.Ht) tiles = (long long)W * H >= 8LL * D.Ws * D.Ht ? 4 : 0;
        if (sp_tiles || cs_tiles) tiles = 0;
        if (tiles >= 0) {
            void *scratch = nullptr;
            cudaMemPool_t pool;
            CU(h, scratch_pool(&pool));
            CU(h, cudaMallocFromPoolAsync(&scratch, render_tiles_scratch_bytes(n_views, W, H), pool, st));
            const cudaError_t e = launch_render_tiles(D, cams, n_views, W, H, d_out, scratch, st, &nl, tiles);
            cudaFreeAsync(scratch, st);
            CU(h, e);
        } else {
            CU(h, launch_render_cta(D, cams, n_views, W, H, d_out, st, &nl, rv >= 6 ? rv - 6 : -1));
        }
    }
    h->launches += nl;
    return HMLFC_OK;
}

int hmlfc_render(const hmlfc_handle *h, const hmlfc_camera *d_cameras, int n_views, int W, int H, uint8_t *d_out,
                 void *cuda_stream)
{
    if (!h) return HMLFC_E_INVALID;
    return render_impl(h, h->ds, d_cameras, n_views, W, H, d_out, cuda_stream);
}

int hmlfc_render_noalloc(const hmlfc_handle *h, const hmlfc_camera *d_cameras, int n_views, int W, int H, uint8_t *d_out,
                         void *cuda_stream)
{
    if (!h || n_views < 0 || W <= 0 || H <= 0 || n_views > 65535 || (n_views > 0 && (!d_cameras || !d_out))) return HMLFC_E_INVALID;
    const DevStream &D = h->ds;
    // streams whose hmlfc_render takes the tile kernels: 4 x 4 blocks; chroma-subsampled or half-pel (not both, windows up to 63) included
    if (D.B != 4 || (D.cs && D.sp) || (D.sp && D.mv_off > 127)) return HMLFC_E_UNSUPPORTED;
    int nl = 0;
    bool too_large = false;
    // tile shape as the automatic choice of hmlfc_render makes it where it takes the tile kernels (32 x 32 for chroma / half-pel streams)
    const int config = (!D.cs && !D.sp && (long long)W * H >= 8LL * D.Ws * D.Ht) ? 4 : 0;
    CU(h, launch_render_tiles_noalloc(D, reinterpret_cast<const Camera *>(d_cameras), n_views, W, H, d_out,
                                      static_cast<cudaStream_t>(cuda_stream), &nl, config, &too_large));
    if (too_large) return HMLFC_E_LIMIT;
    h->launches += nl;
    return HMLFC_OK;
}

int hmlfc_render_lod(const hmlfc_handle *h, const hmlfc_camera *d_cameras, const int32_t *h_levels, int n_views, int W, int H,
                     uint8_t *d_out, void *cuda_stream)
{
    if (!h || n_views < 0 || W <= 0 || H <= 0 || (n_views > 0 && (!d_cameras || !d_out || !h_levels))) return HMLFC_E_INVALID;
    for (int k = 0; k < n_views; ++k)
        if (h_levels[k] < 0 || h_levels[k] > h->ds.h) return HMLFC_E_INVALID;
    // one launch per run of consecutive views with the same level: the kernels take the level from the stream view
    for (int k0 = 0; k0 < n_views;) {
        int k1 = k0 + 1;
        while (k1 < n_views && h_levels[k1] == h_levels[k0]) ++k1;
        DevStream D = h->ds;
        D.lmin = h_levels[k0] > D.lmin ? h_levels[k0] : D.lmin;
        const int rc = render_impl(h, D, d_cameras + k0, k1 - k0, W, H, d_out + (size_t)k0 * (size_t)W * (size_t)H * 3u, cuda_stream);
        if (rc != HMLFC_OK) return rc;
        k0 = k1;
    }
    return HMLFC_OK;
}

int hmlfc_lod_levels(const hmlfc_handle *h, const hmlfc_camera *h_cameras, int n_views, float d0, int32_t *h_levels)
{
    if (!h || n_views < 0 || (n_views > 0 && (!h_cameras || !h_levels))) return HMLFC_E_INVALID;
    for (int k = 0; k < n_views; ++k) {
        const float d = std::fabs(h->ds.z_st - h_cameras[k].eye[2]);
        int L = 0;
        if (d0 > 0.0f)
            while (L < h->ds.h && d >= d0 * (float)(2 << L)) ++L;
        h_levels[k] = L;
    }
    return HMLFC_OK;
}

static int ensure(hmlfc_handle *h, void **buf, size_t *cap, size_t need)
{
    if (need <= *cap) return HMLFC_OK;
    if (*buf) cudaFree(*buf);
    *buf = nullptr; *cap = 0;
    cudaError_t e = cudaMalloc(buf, need);
    if (e != cudaSuccess) { h->last_cuda_error.store((int)e); return e == cudaErrorMemoryAllocation ? HMLFC_E_NOMEM : HMLFC_E_CUDA; }
    *cap = need;
    return HMLFC_OK;
}

// The *_host entry points pipeline their work in chunks over three streams: chunk c+1's input copy (in_stream), chunk c's
// kernel (host_stream) and chunk c-1's result copy (out_stream) overlap, so a call costs about max(copy, kernel) instead of
// their sum.  The bytes written are those of one whole-batch launch (every coordinate / view is independent).
static int sync_pipeline(hmlfc_handle *h)
{
    CU(h, cudaStreamSynchronize(h->out_stream));
    CU(h, cudaStreamSynchronize(h->host_stream));
    CU(h, cudaStreamSynchronize(h->in_stream));
    return HMLFC_OK;
}

int hmlfc_decode_host(hmlfc_handle *h, const int32_t *h_coords, int64_t n, uint8_t *h_out)
{
    if (!h || n < 0 || (n > 0 && (!h_coords || !h_out))) return HMLFC_E_INVALID;
    if (n == 0) return HMLFC_OK;
    int rc;
    if ((rc = ensure(h, &h->d_in, &h->d_in_cap, (size_t)n * 16)) != HMLFC_OK) return rc;
    if ((rc = ensure(h, reinterpret_cast<void **>(&h->d_outbuf), &h->d_out_cap, (size_t)n * 3 + 4)) != HMLFC_OK) return rc;
    // chunks of >= 2^20 coordinates (16 MB in, 3 MB out), a multiple of 1024 so that every chunk's output stays 16-byte aligned
    int64_t chunk = (n + hmlfc_handle::kMaxChunks - 1) / hmlfc_handle::kMaxChunks;
    if (chunk < (1 << 20)) chunk = 1 << 20;
    chunk = (chunk + 1023) / 1024 * 1024;
    const int32_t *d_in = static_cast<const int32_t *>(h->d_in);
    int c = 0;
    for (int64_t i = 0; i < n; i += chunk, ++c) {
        const int64_t m = (n - i < chunk) ? n - i : chunk;
        CU(h, cudaMemcpyAsync(const_cast<int32_t *>(d_in) + i * 4, h_coords + i * 4, (size_t)m * 16, cudaMemcpyHostToDevice, h->in_stream));
        CU(h, cudaEventRecord(h->ev_in[c], h->in_stream));
        CU(h, cudaStreamWaitEvent(h->host_stream, h->ev_in[c], 0));
        if ((rc = hmlfc_decode(h, d_in + i * 4, m, h->d_outbuf + i * 3, h->host_stream)) != HMLFC_OK) { sync_pipeline(h); return rc; }
        CU(h, cudaEventRecord(h->ev_done[c], h->host_stream));
        CU(h, cudaStreamWaitEvent(h->out_stream, h->ev_done[c], 0));
        CU(h, cudaMemcpyAsync(h_out + i * 3, h->d_outbuf + i * 3, (size_t)m * 3, cudaMemcpyDeviceToHost, h->out_stream));
    }
    return sync_pipeline(h);
}

int hmlfc_decode_views_host(hmlfc_handle *h, const int32_t *h_views, int64_t n_views, uint8_t *h_out)
{
    if (!h || n_views < 0 || (n_views > 0 && (!h_views || !h_out))) return HMLFC_E_INVALID;
    if (n_views == 0) return HMLFC_OK;
    const size_t view_bytes = (size_t)h->ds.Ws * h->ds.Ht * 3;
    int rc;
    if ((rc = ensure(h, &h->d_in, &h->d_in_cap, (size_t)n_views * 8)) != HMLFC_OK) return rc;
    if ((rc = ensure(h, reinterpret_cast<void **>(&h->d_outbuf), &h->d_out_cap, (size_t)n_views * view_bytes + 4)) != HMLFC_OK) return rc;
    // chunks of whole views, about 6 MB of pixels each; kernels alternate between two streams, result copies on a third
    int64_t per = (int64_t)((((size_t)6 << 20) + view_bytes - 1) / view_bytes);
    if ((n_views + per - 1) / per > hmlfc_handle::kMaxChunks) per = (n_views + hmlfc_handle::kMaxChunks - 1) / hmlfc_handle::kMaxChunks;
    const int32_t *d_views = static_cast<const int32_t *>(h->d_in);
    CU(h, cudaMemcpyAsync(h->d_in, h_views, (size_t)n_views * 8, cudaMemcpyHostToDevice, h->host_stream));
    CU(h, cudaEventRecord(h->ev_in[0], h->host_stream));
    CU(h, cudaStreamWaitEvent(h->in_stream, h->ev_in[0], 0));
    int c = 0;
    for (int64_t v = 0; v < n_views; v += per, ++c) {
        const int64_t m = (n_views - v < per) ? n_views - v : per;
        cudaStream_t ks = (c & 1) ? h->in_stream : h->host_stream;
        if ((rc = hmlfc_decode_views(h, d_views + 2 * v, m, h->d_outbuf + (size_t)v * view_bytes, ks)) != HMLFC_OK) { sync_pipeline(h); return rc; }
        CU(h, cudaEventRecord(h->ev_done[c], ks));
        CU(h, cudaStreamWaitEvent(h->out_stream, h->ev_done[c], 0));
        CU(h, cudaMemcpyAsync(h_out + (size_t)v * view_bytes, h->d_outbuf + (size_t)v * view_bytes, (size_t)m * view_bytes, cudaMemcpyDeviceToHost, h->out_stream));
    }
    return sync_pipeline(h);
}

int hmlfc_render_host(hmlfc_handle *h, const hmlfc_camera *h_cameras, int n_views, int W, int H, uint8_t *h_out)
{
    if (!h || n_views < 0 || W <= 0 || H <= 0 || (n_views > 0 && (!h_cameras || !h_out))) return HMLFC_E_INVALID;
    if (n_views == 0) return HMLFC_OK;
    const size_t view_bytes = (size_t)W * H * 3;
    const size_t out_bytes = (size_t)n_views * view_bytes;
    int rc;
    if ((rc = ensure(h, &h->d_in, &h->d_in_cap, (size_t)n_views * sizeof(hmlfc_camera))) != HMLFC_OK) return rc;
    if ((rc = ensure(h, reinterpret_cast<void **>(&h->d_outbuf), &h->d_out_cap, out_bytes + 4)) != HMLFC_OK) return rc;
    // Chunks of whole views, about 6 MB of output and at least 2048 tiles (several waves of CTAs) each; batches below 12 MB go
    // as one launch (the copy is short and small launches have a longer tail).  Measured on cfg2 (64 views of 512 x 512 = 50 MB
    // per call; bare copy 0.93 ms, kernel 0.86 ms): one launch 1.79 ms, 6 MB chunks 1.20 ms, 3 MB 1.37 ms, 0.75 MB 1.92 ms
    // (host-side enqueue cost per chunk); cfg3 (16 views = 12.6 MB, kernel 0.97 ms) is slower in chunks.  With the chunks' kernels
    // alternating between two streams (below): cfg2 1.09 ms, cfg4 (16 views of 1024 x 1024) 1.50 -> 1.21 ms, cfg3 in two chunks
    // 1.06 -> 0.96 ms.
    const size_t tiles = (size_t)((W + 31) / 32) * (size_t)((H + 31) / 32);
    size_t per = (((size_t)6 << 20) + view_bytes - 1) / view_bytes;
    if (per * tiles < 2048) per = (2048 + tiles - 1) / tiles;
    if (out_bytes < ((size_t)12 << 20)) per = (size_t)n_views;
    if (((size_t)n_views + per - 1) / per > (size_t)hmlfc_handle::kMaxChunks) per = ((size_t)n_views + hmlfc_handle::kMaxChunks - 1) / hmlfc_handle::kMaxChunks;
    const hmlfc_camera *d_cams = static_cast<const hmlfc_camera *>(h->d_in);
    CU(h, cudaMemcpyAsync(h->d_in, h_cameras, (size_t)n_views * sizeof(hmlfc_camera), cudaMemcpyHostToDevice, h->host_stream));
    // the chunks' kernels alternate between two streams, so the last, partial wave of CTAs of one chunk overlaps the first of the next
    CU(h, cudaEventRecord(h->ev_in[0], h->host_stream));
    CU(h, cudaStreamWaitEvent(h->in_stream, h->ev_in[0], 0));
    int c = 0;
    for (int v = 0; v < n_views; v += (int)per, ++c) {
        const int m = (n_views - v < (int)per) ? n_views - v : (int)per;
        cudaStream_t ks = (c & 1) ? h->in_stream : h->host_stream;
        if ((rc = hmlfc_render(h, d_cams + v, m, W, H, h->d_outbuf + (size_t)v * view_bytes, ks)) != HMLFC_OK) { sync_pipeline(h); return rc; }
        CU(h, cudaEventRecord(h->ev_done[c], ks));
        CU(h, cudaStreamWaitEvent(h->out_stream, h->ev_done[c], 0));
        CU(h, cudaMemcpyAsync(h_out + (size_t)v * view_bytes, h->d_outbuf + (size_t)v * view_bytes, (size_t)m * view_bytes, cudaMemcpyDeviceToHost, h->out_stream));
    }
    return sync_pipeline(h);
}

int hmlfc_last_oob_count(const hmlfc_handle *h, int64_t *out)
{
    if (!h || !out) return HMLFC_E_INVALID;
    unsigned long long v = 0;
    CU(h, cudaDeviceSynchronize());
    CU(h, cudaMemcpy(&v, h->d_oob, sizeof(v), cudaMemcpyDeviceToHost));
    *out = (int64_t)v;
    return HMLFC_OK;
}

static int footprint_common(hmlfc_handle *h, const hmlfc_camera *d_cameras, int n_views, int W, int H, const int32_t *d_coords,
                            int64_t n, hmlfc_footprint_t *out)
{
    const DevStream &D = h->ds;
    if (D.cs || D.sp) return HMLFC_E_UNSUPPORTED;  // the counting kernels (a measurement aid) assume one block grid for the three channels and one reference sample per tap
    const size_t blk_words = ((size_t)h->n_pc * (size_t)D.nblk + 31) / 32 + 1;
    const size_t rkv_words = ((size_t)D.UH * D.VH * D.Ht * D.Ws + 31) / 32 + 1;
    FootprintMarks mk{nullptr, nullptr};
    FootprintTotals *d_tot = nullptr, tot{};
    int rc = HMLFC_OK;
    cudaError_t e;
    if ((e = cudaMalloc(reinterpret_cast<void **>(&mk.blk), blk_words * 4)) != cudaSuccess ||
        (e = cudaMalloc(reinterpret_cast<void **>(&mk.rkv), rkv_words * 4)) != cudaSuccess ||
        (e = cudaMalloc(reinterpret_cast<void **>(&d_tot), sizeof(FootprintTotals))) != cudaSuccess ||
        (e = cudaMemset(mk.blk, 0, blk_words * 4)) != cudaSuccess || (e = cudaMemset(mk.rkv, 0, rkv_words * 4)) != cudaSuccess ||
        (e = cudaMemset(d_tot, 0, sizeof(FootprintTotals))) != cudaSuccess ||
        (e = d_cameras ? launch_footprint_render(D, reinterpret_cast<const Camera *>(d_cameras), n_views, W, H, mk, nullptr)
                       : launch_footprint_decode(D, d_coords, n, mk, nullptr)) != cudaSuccess ||
        (e = launch_footprint_reduce(D, h->n_pc, h->d_bits15, h->mv_bits15, mk, d_tot, nullptr)) != cudaSuccess ||
        (e = cudaMemcpy(&tot, d_tot, sizeof(tot), cudaMemcpyDeviceToHost)) != cudaSuccess)
        rc = cuda_fail(h, e);
    cudaFree(mk.blk); cudaFree(mk.rkv); cudaFree(d_tot);
    if (rc != HMLFC_OK) return rc;
    out->blocks_touched = (int64_t)tot.blocks;
    out->flag_bits = (int64_t)tot.flag_bits;
    out->payload_bits15 = (int64_t)tot.payload_bits15;
    out->mv_bits15 = (int64_t)tot.mv_bits15;
    out->rkv_bytes = (int64_t)tot.rkv_samples * 5;  // Y 1 byte + Co, Cg 2 bytes each
    if (d_cameras) { out->out_bytes = (int64_t)n_views * W * H * 3; out->in_bytes = (int64_t)n_views * 64; }
    else { out->out_bytes = n * 3; out->in_bytes = n * 16; }
    out->bytes_alg = ((double)out->flag_bits + (double)(out->payload_bits15 + out->mv_bits15) / 15.0) / 8.0 +
                     (double)out->rkv_bytes + (double)out->out_bytes + (double)out->in_bytes;
    return HMLFC_OK;
}

int hmlfc_footprint_render(hmlfc_handle *h, const hmlfc_camera *d_cameras, int n_views, int W, int H, hmlfc_footprint_t *out)
{
    if (!h || !out || !d_cameras || n_views <= 0 || n_views > 65535 || W <= 0 || H <= 0) return HMLFC_E_INVALID;
    return footprint_common(h, d_cameras, n_views, W, H, nullptr, 0, out);
}

int hmlfc_footprint_decode(hmlfc_handle *h, const int32_t *d_coords, int64_t n, hmlfc_footprint_t *out)
{
    if (!h || !out || !d_coords || n <= 0) return HMLFC_E_INVALID;
    return footprint_common(h, nullptr, 0, 0, 0, d_coords, n, out);
}

int hmlfc_set_render_variant(hmlfc_handle *h, int variant)
{
    if (!h || variant < 0 || variant > 15 || variant == 2 || variant == 3) return HMLFC_E_INVALID;  // 2, 3: removed kernels
    h->render_variant = variant;
    return HMLFC_OK;
}

int hmlfc_set_min_level(hmlfc_handle *h, int min_level)
{
    if (!h || min_level < 0 || min_level > h->ds.h) return HMLFC_E_INVALID;
    h->ds.lmin = min_level;
    return HMLFC_OK;
}

int hmlfc_set_decode_variant(hmlfc_handle *h, int variant)
{
    if (!h || variant < 0 || variant > 4) return HMLFC_E_INVALID;
    h->decode_variant = variant;
    return HMLFC_OK;
}

int hmlfc_launch_count(const hmlfc_handle *h, int64_t *out)
{
    if (!h || !out) return HMLFC_E_INVALID;
    *out = h->launches.load();
    return HMLFC_OK;
}

int hmlfc_last_cuda_error(const hmlfc_handle *h) { return h ? h->last_cuda_error.load() : 0; }

void hmlfc_free(hmlfc_handle *h) { release(h); }

}  // extern "C"
