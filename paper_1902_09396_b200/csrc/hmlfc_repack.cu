// hmlfc_load, device side: the block records of a stream (hmlfc_device.cuh, "block records").
//
// The serialized HMLFC stream stores one BISE string of values per plane-channel and one of motion records
// (PAPER.md:272); a random sample therefore gathers its plane's contribution from up to six unrelated sectors.  This
// kernel decodes every stored value and motion record once, right after the upload, and writes them back grouped per block as plain
// binary fields.  The codes are copied, not interpreted: what the decoders compute from them is unchanged.
#include "hmlfc_kernels.cuh"

namespace hmlfc {

namespace {

// OR the w-bit field v into brec[] at bit `bit` (records of neighbouring blocks share words: atomics; the array starts zeroed)
__device__ __forceinline__ void put_field(uint32_t *__restrict__ brec, unsigned long long bit, uint32_t w, uint32_t v)
{
    if (w == 0u) return;
    const unsigned long long wi = bit >> 5;
    const uint32_t sh = (uint32_t)bit & 31u;
    atomicOr(brec + wi, v << sh);
    if (sh + w > 32u) atomicOr(brec + wi + 1, v >> (32u - sh));
}

// one thread per (plane, block)
__global__ void __launch_bounds__(256)
repack_kernel(const DevStream S, unsigned long long n_items, uint32_t *__restrict__ brec)
{
    const unsigned long long i = (unsigned long long)blockIdx.x * 256ull + threadIdx.x;
    if (i >= n_items) return;
    const uint32_t p = (uint32_t)(i / (unsigned long long)S.nblk), b = (uint32_t)(i - (unsigned long long)p * S.nblk);
    const uint32_t g = b >> 5, bit = 1u << (b & 31);
    const uint4 *slot = S.bslot + ((size_t)p * (size_t)S.fgroups + (size_t)g) * 2u;
    const uint4 sa = ldg(slot), sb = ldg(slot + 1);
    if (!((sa.x | sa.y | sa.z | sa.w | sb.x | sb.y) & bit)) return;
    uint4 fr[3];  // the ranks: where the block's values and motion record are in the stream's own strings
#pragma unroll
    for (int c = 0; c < 3; ++c) fr[c] = ldg(S.flagrec + flag_index(S, 3u * p + (uint32_t)c, g));
    const uint4 pb = ldg(S.pb + p);
    const BrecPos r = brec_locate(S, sa, sb, bit, pb);
    const uint32_t BB = 1u << (2 * S.logB);
#pragma unroll 1
    for (int c = 0; c < 3; ++c) {
        const uint4 d = ldg(S.pc + 3u * p + (uint32_t)c);
        if (r.pred & (1u << c)) {
            const uint32_t mi = fr[c].w + popc(fr[c].z & (bit - 1u));
            put_field(brec, r.bit + brec_mv_offset(r, pb, c), pb.y >> 24, bise_decode_at(S.mv + d.z, mi, S.mv_layout, S.mv_m));
        }
        if (r.res & (1u << c)) {
            const uint32_t rank = fr[c].y + popc(fr[c].x & (bit - 1u)), w = (pb.y >> (8 * c)) & 0xFFu;
            for (uint32_t k = 0; k < BB; ++k)
                put_field(brec, r.bit + brec_sample_offset(r, pb, k) + brec_channel_offset(r, pb, c), w, bise_decode_at(S.pay + d.y, rank * BB + k, pc_layout(d.w), pc_m(d.w)));
        }
    }
}

}  // namespace

// S.pb and the stream's other arrays are on the device; d_brec (zeroed by the caller) receives the block records
cudaError_t launch_repack(const DevStream &S, uint64_t n_planes, uint32_t *d_brec, cudaStream_t st)
{
    const unsigned long long n_items = (unsigned long long)n_planes * (unsigned long long)S.nblk;
    if (n_items == 0) return cudaSuccess;
    const unsigned long long blocks = (n_items + 255) / 256;
    if (blocks > 0x7fffffffull) return cudaErrorInvalidValue;
    repack_kernel<<<(unsigned)blocks, 256, 0, st>>>(S, n_items, d_brec);
    return cudaGetLastError();
}

}  // namespace hmlfc
