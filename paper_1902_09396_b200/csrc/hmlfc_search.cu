// hmlfc_search: phase-shifted exhaustive block motion search of the HMLFC encoder on sm_100a.
//
// PAPER.md:227-248, Eqs. (1)-(2): for every block B_P of a predictive SRV image P and every motion vector (x,y) in
// [-W,W]^2 of its cluster's reference SRV image R,
//     Delta-(x,y) = sum_l |B_P(l) - B_R^{xy}(l)| ,   Delta+(x,y) = sum_l |B_P(l) + B_R^{xy}(l)| ,
//     Delta = min(min_xy Delta-, min_xy Delta+)  with the motion vector and the mode (subtractive / additive =
//     "phase-shifted") of the minimum.   PAPER.md:387: this search is why encoding takes 30-90 minutes on a CPU.
// Readings (R8, R9): R reads 0 outside the image; ties: subtractive before additive, then the smallest dy,
// then the smallest dx -- i.e. the minimum of the key (SAD, mode, dy, dx) in lexicographic order.
//
// The arithmetic is fp32 on purpose: every operand is an integer of magnitude <= 65534 and every sum stays below
// 2^24, so fp32 adds are exact, |x| is a free source modifier of FADD, and the FP32 pipe has twice the lanes of the
// INT32 pipe on this SM.  The result is bit-identical to the integer definition.
//
// One CTA searches a tile of 8 x 8 blocks of one (P, R) pair.  The reference window of the tile (tile + W on every
// side, zero outside the image) and the tile of P are staged in shared memory as floats.  A task = (block, dy, chunk
// of 12 consecutive dx): the thread reads, per block row, 16 consecutive window samples with four 128-bit shared
// loads and updates 12 + 12 running sums held in registers (192 FADDs per 4 shared loads).  Tasks are ordered
// (chunk, dy, block): a warp's lanes work on 32 neighbouring blocks at one (dy, chunk) -- consecutive 128-bit loads --
// and every task of a thread belongs to one block, whose minimum key the thread keeps in registers.  Block sizes
// other than 4 take a plain warp-per-block kernel.
#include <cuda_runtime.h>
#include <stdint.h>

#include "hmlfc.h"

namespace hmlfc {

namespace {

constexpr int kTBX = 8, kTBY = 8;  // blocks per CTA tile
constexpr int kChunk = 12;         // dx offsets per task
constexpr int kThreads = 256;

__host__ __device__ inline int window_stride(int W)
{
    const int nchunks = (2 * W + 1 + kChunk - 1) / kChunk;
    const int need = (kTBX - 1) * 4 + (nchunks - 1) * kChunk + 16;  // the 16-sample read of the last block's last chunk ends here
    return ((need - 4 + 31) / 32) * 32 + 4;                         // smallest stride >= need that is 4 mod 32
}

__device__ __forceinline__ unsigned long long make_key(float sad, int mode, int dyi, int dxi)
{
    return ((unsigned long long)(unsigned)__float2int_rn(sad) << 32) | ((unsigned long long)mode << 16) |
           ((unsigned long long)dyi << 8) | (unsigned long long)dxi;
}

// One task: the block's 4 x 4 samples against NOFF consecutive dx offsets at one dy, both modes; returns the task's minimum key in
// the order (SAD, mode, dx): subtractive sums first, strict comparisons keep the first (offset 0 of a chunk always exists).
// NOFF + 3 window samples per row come from (NOFF + 3 + 3) / 4 128-bit shared loads.
template <int NOFF>
__device__ __forceinline__ unsigned long long task_min(const float *__restrict__ prow, const float *__restrict__ wrow, int stride, int nvalid,
                                                       int dyi, int chunk)
{
    constexpr int NLD = (NOFF + 3 + 3) / 4;
    float sm[NOFF], sp[NOFF];
#pragma unroll
    for (int d = 0; d < NOFF; ++d) sm[d] = sp[d] = 0.f;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const float4 p4 = *reinterpret_cast<const float4 *>(prow + j * (kTBX * 4));
        const float p[4] = {p4.x, p4.y, p4.z, p4.w};
        const float4 *row = reinterpret_cast<const float4 *>(wrow + (size_t)j * stride);
        float r[4 * NLD];
#pragma unroll
        for (int q = 0; q < NLD; ++q) {
            const float4 v = row[q];
            r[4 * q + 0] = v.x; r[4 * q + 1] = v.y; r[4 * q + 2] = v.z; r[4 * q + 3] = v.w;
        }
#pragma unroll
        for (int d = 0; d < NOFF; ++d)
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                sm[d] += fabsf(p[i] - r[d + i]);  // Eq. (1)
                sp[d] += fabsf(p[i] + r[d + i]);  // Eq. (2)
            }
    }
    float bs = sm[0];
    int bi = 0;
#pragma unroll
    for (int d = 1; d < NOFF; ++d)
        if (d < nvalid && sm[d] < bs) { bs = sm[d]; bi = d; }
#pragma unroll
    for (int d = 0; d < NOFF; ++d)
        if (d < nvalid && sp[d] < bs) { bs = sp[d]; bi = 16 + d; }
    return make_key(bs, bi >> 4, dyi, chunk * kChunk + (bi & 15));
}

#ifndef HMLFC_SEARCH_MINB
#define HMLFC_SEARCH_MINB 4
#endif
__global__ void __launch_bounds__(kThreads, HMLFC_SEARCH_MINB)
search4_kernel(const int16_t *__restrict__ planes, const int2 *__restrict__ pairs, int Ws, int Ht, int W, int nbx, int nby,
               int4 *__restrict__ out)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int nd = 2 * W + 1, nchunks = (nd + kChunk - 1) / kChunk;
    const int stride = window_stride(W), wrows = kTBY * 4 + 2 * W;
    float *win = reinterpret_cast<float *>(smem_raw);                                  // [wrows][stride]
    float *ptile = win + (size_t)wrows * stride;                                       // [kTBY*4][kTBX*4]
    unsigned long long *best = reinterpret_cast<unsigned long long *>(ptile + kTBY * 4 * kTBX * 4);  // [kTBY*kTBX]

    const int tid = threadIdx.x;
    const int2 pr = pairs[blockIdx.z];
    const int16_t *P = planes + (size_t)pr.x * (size_t)Ws * (size_t)Ht;
    const int16_t *R = planes + (size_t)pr.y * (size_t)Ws * (size_t)Ht;
    const int x0 = blockIdx.x * kTBX * 4, y0 = blockIdx.y * kTBY * 4;

    // stage the reference window (zero outside the image, R8), the tile of P, and reset the minima
    for (int q = tid; q < wrows * stride; q += kThreads) {
        const int wy = q / stride, wx = q - wy * stride;
        const int gx = x0 - W + wx, gy = y0 - W + wy;
        float v = 0.f;
        if ((unsigned)gx < (unsigned)Ws && (unsigned)gy < (unsigned)Ht) v = (float)R[(size_t)gy * Ws + gx];
        win[q] = v;
    }
    for (int q = tid; q < kTBY * 4 * kTBX * 4; q += kThreads) {
        const int py = q / (kTBX * 4), px = q - py * (kTBX * 4);
        const int gx = x0 + px, gy = y0 + py;
        ptile[q] = (gx < Ws && gy < Ht) ? (float)P[(size_t)gy * Ws + gx] : 0.f;
    }
    if (tid < kTBX * kTBY) best[tid] = ~0ull;
    __syncthreads();

    // Tasks in the order (chunk, dy, block): the 32 lanes of a warp work on the tile's 32 blocks at one (dy, chunk), so the chunk --
    // and with it the number of valid offsets -- is warp-uniform.  The last chunk holds nd - 12 (nchunks - 1) offsets (9 for W = 16):
    // it runs the same body instantiated for 9 offsets and 12 window samples instead of computing 12 and discarding 3.
    const int per_chunk = kTBX * kTBY * nd, ntasks = per_chunk * nchunks;
    const int nlast = nd - (nchunks - 1) * kChunk;
    // kThreads is a multiple of the 32 blocks of a tile: all tasks of a thread belong to ONE block (blk = tid mod 32), so the thread
    // keeps its minimum key in registers and publishes it once
    static_assert(kThreads % (kTBX * kTBY) == 0, "a thread's tasks must stay on one block");
    unsigned long long kbest = ~0ull;
    for (int t = tid; t < ntasks; t += kThreads) {
        const int chunk = t / per_chunk, rem = t - chunk * per_chunk;
        const int dyi = rem / (kTBX * kTBY), blk = rem - dyi * (kTBX * kTBY);
        const int bxl = blk & (kTBX - 1), byl = blk / kTBX;
        if (blockIdx.x * kTBX + bxl >= nbx || blockIdx.y * kTBY + byl >= nby) continue;
        const float *prow = ptile + (byl * 4) * (kTBX * 4) + bxl * 4;
        // window row of image row y0 + byl*4 + j + dy; column of image column x0 + bxl*4 + dx, dx = chunk*12 - W + d
        const float *wrow = win + (size_t)(byl * 4 + dyi) * stride + bxl * 4 + chunk * kChunk;
        unsigned long long k;
        if (chunk == nchunks - 1 && nlast == 9) k = task_min<9>(prow, wrow, stride, 9, dyi, chunk);
        else k = task_min<kChunk>(prow, wrow, stride, chunk == nchunks - 1 ? nlast : kChunk, dyi, chunk);
        kbest = k < kbest ? k : kbest;
    }
    if (kbest != ~0ull) atomicMin(&best[tid & (kTBX * kTBY - 1)], kbest);
    __syncthreads();
    if (tid < kTBX * kTBY) {
        const int bx = blockIdx.x * kTBX + (tid & (kTBX - 1)), by = blockIdx.y * kTBY + tid / kTBX;
        if (bx < nbx && by < nby) {
            const unsigned long long k = best[tid];
            out[((size_t)blockIdx.z * nby + by) * nbx + bx] =
                make_int4((int)((k >> 16) & 1u), (int)(k & 0xFFu) - W, (int)((k >> 8) & 0xFFu) - W, (int)(k >> 32));
        }
    }
}

// any block size: one warp per block, lanes stride over the (dy, dx) offsets, samples straight from global memory
__global__ void __launch_bounds__(kThreads)
search_generic_kernel(const int16_t *__restrict__ planes, const int2 *__restrict__ pairs, int n_pairs, int Ws, int Ht, int B, int W,
                      int nbx, int nby, int4 *__restrict__ out)
{
    const int lane = threadIdx.x & 31;
    const long long wid = (long long)blockIdx.x * (kThreads / 32) + (threadIdx.x >> 5);
    const long long nblk = (long long)nbx * nby;
    if (wid >= nblk * n_pairs) return;
    const int pair = (int)(wid / nblk), b = (int)(wid - (long long)pair * nblk);
    const int by = b / nbx, bx = b - by * nbx;
    const int2 pr = pairs[pair];
    const int16_t *P = planes + (size_t)pr.x * (size_t)Ws * (size_t)Ht;
    const int16_t *R = planes + (size_t)pr.y * (size_t)Ws * (size_t)Ht;
    const int nd = 2 * W + 1;
    unsigned long long k = ~0ull;
    for (int o = lane; o < nd * nd; o += 32) {
        const int dyi = o / nd, dxi = o - dyi * nd;
        float sm = 0.f, sp = 0.f;
        for (int j = 0; j < B; ++j)
            for (int i = 0; i < B; ++i) {
                const int x = bx * B + i, y = by * B + j, rx = x + dxi - W, ry = y + dyi - W;
                const float p = (float)P[(size_t)y * Ws + x];
                const float r = ((unsigned)rx < (unsigned)Ws && (unsigned)ry < (unsigned)Ht) ? (float)R[(size_t)ry * Ws + rx] : 0.f;
                sm += fabsf(p - r);
                sp += fabsf(p + r);
            }
        const unsigned long long km = make_key(sm, 0, dyi, dxi), kp = make_key(sp, 1, dyi, dxi);
        k = km < k ? km : k;
        k = kp < k ? kp : k;
    }
    for (int o = 16; o > 0; o >>= 1) {
        const unsigned long long other = __shfl_xor_sync(0xffffffffu, k, o);
        k = other < k ? other : k;
    }
    if (lane == 0)
        out[(size_t)pair * nblk + b] = make_int4((int)((k >> 16) & 1u), (int)(k & 0xFFu) - W, (int)((k >> 8) & 0xFFu) - W, (int)(k >> 32));
}

}  // namespace

}  // namespace hmlfc

extern "C" int hmlfc_search(const int16_t *d_planes, const int32_t *d_pairs, int n_pairs, int Ws, int Ht, int block, int window,
                            int32_t *d_out, void *cuda_stream)
{
    using namespace hmlfc;
    if (n_pairs < 0 || Ws <= 0 || Ht <= 0 || (n_pairs > 0 && (!d_planes || !d_pairs || !d_out))) return HMLFC_E_INVALID;
    if (block < 1 || block > 8 || window < 0 || window > 64 || Ws % block || Ht % block) return HMLFC_E_UNSUPPORTED;
    if (n_pairs == 0) return HMLFC_OK;
    if (n_pairs > 65535) return HMLFC_E_UNSUPPORTED;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const int nbx = Ws / block, nby = Ht / block;
    const int2 *pairs = reinterpret_cast<const int2 *>(d_pairs);
    int4 *out = reinterpret_cast<int4 *>(d_out);
    if (block == 4) {
        const size_t smem = ((size_t)(kTBY * 4 + 2 * window) * window_stride(window) + kTBY * 4 * kTBX * 4) * sizeof(float) +
                            kTBX * kTBY * sizeof(unsigned long long);
        if (smem > 48 * 1024 &&
            cudaFuncSetAttribute(search4_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
            return HMLFC_E_CUDA;
        dim3 grid((unsigned)((nbx + kTBX - 1) / kTBX), (unsigned)((nby + kTBY - 1) / kTBY), (unsigned)n_pairs);
        if (grid.y > 65535u) return HMLFC_E_UNSUPPORTED;
        search4_kernel<<<grid, kThreads, smem, st>>>(d_planes, pairs, Ws, Ht, window, nbx, nby, out);
    } else {
        const long long warps = (long long)nbx * nby * n_pairs;
        const long long blocks = (warps + kThreads / 32 - 1) / (kThreads / 32);
        if (blocks > 0x7fffffffLL) return HMLFC_E_UNSUPPORTED;
        search_generic_kernel<<<(unsigned)blocks, kThreads, 0, st>>>(d_planes, pairs, n_pairs, Ws, Ht, block, window, nbx, nby, out);
    }
    return cudaGetLastError() == cudaSuccess ? HMLFC_OK : HMLFC_E_CUDA;
}
