// gather_probe: what does the B200 memory system deliver for the access pattern of hmlfc_decode -- every lane of a
// warp reading its own random 32-byte sector?  Times `iters` dependent-free gathers per thread from a table of
// `table_bytes` (8 MB: L2-resident, like the cfg2 stream; 1 GB: HBM-resident, like cfg4 / cfg5) with one 32-, 64-,
// 128- or 256-bit load per lane, or 2 x 128 / 4 x 32 bits as separate loads to the same sector.  Measurement aid
// (DESIGN.md 9.4); not on the hot path.  C ABI: hmlfc_gather_probe(mode, table_bytes, &ms, &lane_gathers).
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

__device__ __forceinline__ uint32_t mix(uint32_t x)
{
    x ^= x >> 16; x *= 0x7feb352dU; x ^= x >> 15; x *= 0x846ca68bU; x ^= x >> 16;
    return x;
}

template <int MODE>
__global__ void gather_kernel(const uint32_t *__restrict__ p, uint32_t sector_mask, int iters, uint32_t *out)
{
    const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t acc = 0;
    for (int it = 0; it < iters; ++it) {
        const uint32_t *q = p + (size_t)(mix(t * 977u + it * 0x9e3779b9u) & sector_mask) * 8;  // a random 32-byte sector
        if (MODE == 0) acc += __ldg(q);
        else if (MODE == 1) { const uint2 v = __ldg(reinterpret_cast<const uint2 *>(q)); acc += v.x ^ v.y; }
        else if (MODE == 2) { const uint4 v = __ldg(reinterpret_cast<const uint4 *>(q)); acc += v.x ^ v.y ^ v.z ^ v.w; }
        else if (MODE == 3) {
            const uint4 v = __ldg(reinterpret_cast<const uint4 *>(q)), w = __ldg(reinterpret_cast<const uint4 *>(q) + 1);
            acc += v.x ^ v.y ^ v.z ^ v.w ^ w.x ^ w.y ^ w.z ^ w.w;
        } else if (MODE == 4) {
            uint32_t a0, a1, a2, a3, a4, a5, a6, a7;  // LDG.E.ENL2.256: one 256-bit load per lane (sm_100a)
            asm volatile("ld.global.nc.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                         : "=r"(a0), "=r"(a1), "=r"(a2), "=r"(a3), "=r"(a4), "=r"(a5), "=r"(a6), "=r"(a7) : "l"(q));
            acc += a0 ^ a1 ^ a2 ^ a3 ^ a4 ^ a5 ^ a6 ^ a7;
        } else acc += __ldg(q) ^ __ldg(q + 1) ^ __ldg(q + 2) ^ __ldg(q + 3);
    }
    out[t] = acc;
}

template <int MODE>
cudaError_t run(const uint32_t *d, uint32_t mask, int iters, int blocks, int threads, uint32_t *out, float *ms)
{
    cudaEvent_t a, b;
    cudaEventCreate(&a); cudaEventCreate(&b);
    gather_kernel<MODE><<<blocks, threads>>>(d, mask, iters, out);  // warm-up
    cudaEventRecord(a);
    gather_kernel<MODE><<<blocks, threads>>>(d, mask, iters, out);
    cudaEventRecord(b);
    cudaError_t e = cudaEventSynchronize(b);
    if (e == cudaSuccess) e = cudaEventElapsedTime(ms, a, b);
    cudaEventDestroy(a); cudaEventDestroy(b);
    return e;
}

}  // namespace

// mode: 0 = 32-bit, 1 = 64-bit, 2 = 128-bit, 3 = 2 x 128-bit same sector, 4 = 256-bit, 5 = 4 x 32-bit same sector.
// table_bytes must be a power of two >= 32.  Returns 0 or the cudaError_t.
extern "C" int hmlfc_gather_probe(int mode, unsigned long long table_bytes, float *ms, double *lane_gathers)
{
    if (mode < 0 || mode > 5 || table_bytes < 32 || (table_bytes & (table_bytes - 1)) || !ms || !lane_gathers) return -1;
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int iters = 64, threads = 256, blocks = sms * 16;
    uint32_t *d = nullptr, *out = nullptr;
    cudaError_t e = cudaMalloc(&d, table_bytes);
    if (e != cudaSuccess) return (int)e;
    e = cudaMalloc(&out, (size_t)blocks * threads * 4);
    if (e != cudaSuccess) { cudaFree(d); return (int)e; }
    cudaMemset(d, 1, table_bytes);
    const uint32_t mask = (uint32_t)(table_bytes / 32 - 1);
    switch (mode) {
    case 0: e = run<0>(d, mask, iters, blocks, threads, out, ms); break;
    case 1: e = run<1>(d, mask, iters, blocks, threads, out, ms); break;
    case 2: e = run<2>(d, mask, iters, blocks, threads, out, ms); break;
    case 3: e = run<3>(d, mask, iters, blocks, threads, out, ms); break;
    case 4: e = run<4>(d, mask, iters, blocks, threads, out, ms); break;
    default: e = run<5>(d, mask, iters, blocks, threads, out, ms); break;
    }
    *lane_gathers = (double)blocks * threads * iters;
    cudaFree(d); cudaFree(out);
    return (int)e;
}
