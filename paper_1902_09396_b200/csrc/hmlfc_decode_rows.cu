// hmlfc_decode_views / hmlfc_decode_blocks for B = 4 streams (sm_100a): one lane per block-ROW segment.
//
// PAPER.md:289-293 (decoding procedure), :309 ("As a block of pixels are decoded ..."): definitions in DESIGN.md section 3.
#include "hmlfc_kernels.cuh"
#include "hmlfc_bise_row.cuh"

namespace hmlfc {

namespace {

constexpr int kNT = 256;  // threads per CTA

// ---------------------------------------------------------------------------------------------------------------
// hmlfc_decode_views for B = 4 streams: one lane per block ROW segment (4 consecutive pixels of one block of one view).  The same
// per-row decode as phase B3 -- flag / rank record once per (level, channel), the row's 4 stored values from one pass over two
// 64-bit BISE windows, the motion record once, the motion-compensated reference row from at most two reference blocks -- without
// the shared-memory tables of the render kernel: whole views need no footprint.  PAPER.md:289-293; DESIGN.md section 3.
// kBlocks (hmlfc_decode_blocks): the segments are the 4 rows of arbitrary 4 x 4 blocks (u, v, bx, by) = blocks[g / 4] -- random access at
// the granularity the paper decodes at ("As a block of pixels are decoded ...") -- written as [n][4][4][3].
// kSubpel: streams with half-pel motion offsets (R28): the reference row is the rounded mean of 1 / 2 / 4 samples of up to two rows.
// kCs: chroma-subsampled streams (R18): for Co / Cg the lane decodes the row of the CHROMA block that holds its two chroma samples
// ((s0 >> 1) .. (s0 >> 1) + 1 of row t >> 1) with the channel's own geometry and takes those two (each serves two of its four pixels).
template <bool kBlocks, bool kSubpel = false, bool kCs = false>
__global__ void __launch_bounds__(kNT)
decode_rows_kernel(const __grid_constant__ DevStream S, const int2 *__restrict__ views, long long n_seg, uint8_t *__restrict__ out,
                   unsigned long long *__restrict__ oob, int out_aligned)
{
    __shared__ uint16_t lut[384];
    for (int q = threadIdx.x; q < 192; q += kNT)
        reinterpret_cast<uint32_t *>(lut)[q] = reinterpret_cast<const uint32_t *>(g_cta_digit_lut.v)[q];
    __syncthreads();
    const long long g = (long long)blockIdx.x * kNT + threadIdx.x;
    if (g >= n_seg) return;
    long long view = 0;
    int t, bx, u, v;
    bool in_range;
    if (kBlocks) {
        const int4 q = __ldg(reinterpret_cast<const int4 *>(views) + (g >> 2));
        u = q.x; v = q.y; bx = q.z; t = (q.w << 2) + (int)(g & 3);
        in_range = (unsigned)u < (unsigned)S.U && (unsigned)v < (unsigned)S.V && (unsigned)q.z < (unsigned)S.nbx && (unsigned)q.w < (unsigned)S.nby;
    } else {
        const long long seg_per_view = (long long)S.nbx * S.Ht;
        view = g / seg_per_view;
        const int seg = (int)(g - view * seg_per_view);
        t = seg / S.nbx; bx = seg - t * S.nbx;
        const int2 uv = __ldg(views + view);
        u = uv.x; v = uv.y;
        in_range = (unsigned)u < (unsigned)S.U && (unsigned)v < (unsigned)S.V;
    }
    const int s0 = bx << 2, h = S.h;
    uint32_t rgb[4] = {0u, 0u, 0u, 0u};
    if (in_range) {
        int a[3][4];
        {
            const short4 *r = S.rkv + ((size_t)((v >> h) * S.UH + (u >> h)) * (size_t)S.Ht + (size_t)t) * (size_t)S.Ws + (size_t)s0;
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const short4 k = ldg(r + i);
                a[0][i] = k.x; a[1][i] = k.y; a[2][i] = k.z;
            }
        }
        for (int L = S.lmin; L < h; ++L) {
            const LevelDesc lv = S.lev[L];
            const int pu = u >> L, pv = v >> L;
            const uint32_t pc0 = lv.pc_base + (uint32_t)(pv * lv.UL + pu) * 3u;
            const uint32_t refpc0 = lv.pc_base + (uint32_t)((pv & ~1) * lv.UL + (pu & ~1)) * 3u;
            const bool predictive = ((pu | pv) & 1) != 0;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                // the channel's geometry: row tc of its plane, first sample sc0 of the block row segment, block grid, image height
                const int csh = (kCs && c > 0) ? 1 : 0;
                const int tc = t >> csh, sc0 = csh ? ((s0 >> 1) & ~3) : s0, cnbx = csh ? S.nbx_c : S.nbx, cHt = S.Ht >> csh;
                const int b = (tc >> 2) * cnbx + (sc0 >> 2);
                const uint32_t g32 = (uint32_t)(b >> 5), bit = 1u << (b & 31), i0 = (uint32_t)((tc & 3) << 2);
                const uint4 d = ldg(S.pc + pc0 + c);
                const uint4 fr = ldg(S.flagrec + d.x + 4u * g32);
                uint2 own = make_uint2(0u, 0u);
                if (fr.x & bit) own = bise_row4(S.pay + d.y, ((fr.y + popc(fr.x & (bit - 1u))) << 4) + i0, d.w, lut);
                int e0 = (int)(int16_t)(own.x & 0xFFFFu), e1 = (int)own.x >> 16, e2 = (int)(int16_t)(own.y & 0xFFFFu), e3 = (int)own.y >> 16;
                if (predictive && (fr.z & bit)) {
                    const uint32_t mr = bise_at(S.mv + d.z, fr.w + popc(fr.z & (bit - 1u)), S.mv_layout, S.mv_m, lut);
                    int md, dx, dy;
                    mv_unpack(S, mr, md, dx, dy);
                    if (!kSubpel) {
                        const int rx = sc0 + dx, ry = tc + dy;
                        if ((unsigned)ry < (unsigned)cHt) {
                            const uint4 dr = ldg(S.pc + refpc0 + c);
                            // the 4 reference samples (rx .. rx+3, ry) lie in the block row ry>>2, blocks rx>>2 and (rx>>2)+1
                            const int o = rx & 3, bxa = rx >> 2;
                            const uint32_t j0 = (uint32_t)((ry & 3) << 2);
                            const int rowb = (ry >> 2) * cnbx;
                            uint2 qa = make_uint2(0u, 0u), qb = make_uint2(0u, 0u);
                            if ((unsigned)bxa < (unsigned)cnbx) {
                                const int rb = rowb + bxa;
                                const uint4 rf = ldg(S.flagrec + dr.x + 4u * (uint32_t)(rb >> 5));
                                const uint32_t rbit = 1u << (rb & 31);
                                if (rf.x & rbit) qa = bise_row4(S.pay + dr.y, ((rf.y + popc(rf.x & (rbit - 1u))) << 4) + j0, dr.w, lut);
                            }
                            if (o && (unsigned)(bxa + 1) < (unsigned)cnbx) {
                                const int rb = rowb + bxa + 1;
                                const uint4 rf = ldg(S.flagrec + dr.x + 4u * (uint32_t)(rb >> 5));
                                const uint32_t rbit = 1u << (rb & 31);
                                if (rf.x & rbit) qb = bise_row4(S.pay + dr.y, ((rf.y + popc(rf.x & (rbit - 1u))) << 4) + j0, dr.w, lut);
                            }
                            uint32_t w0 = qa.x, w1 = qa.y, w2 = qb.x, w3 = qb.y;
                            if (o & 2) { w0 = w1; w1 = w2; w2 = w3; }
                            const uint32_t sh = (uint32_t)(o & 1) << 4;
                            const uint32_t q01 = __funnelshift_r(w0, w1, sh), q23 = __funnelshift_r(w1, w2, sh);
                            const int q0 = (int)(int16_t)(q01 & 0xFFFFu), q1 = (int)q01 >> 16, q2 = (int)(int16_t)(q23 & 0xFFFFu), q3 = (int)q23 >> 16;
                            if (md) { e0 -= q0; e1 -= q1; e2 -= q2; e3 -= q3; }   // R10: additive P = e - R
                            else { e0 += q0; e1 += q1; e2 += q2; e3 += q3; }      //      subtractive P = e + R
                        }
                    } else {
                        const int fx = dx & 1, fy = dy & 1;
                        const int rx = sc0 + (dx >> 1), ry = tc + (dy >> 1), o = rx & 3, bxa = rx >> 2;
                        const uint4 dr = ldg(S.pc + refpc0 + c);
                        int h0 = 0, h1 = 0, h2 = 0, h3 = 0;
#pragma unroll
                        for (int jr = 0; jr < 2; ++jr) {
                            const int r = ry + jr;
                            if ((jr && !fy) || (unsigned)r >= (unsigned)cHt) continue;
                            const uint32_t j0 = (uint32_t)((r & 3) << 2);
                            const int rowb = (r >> 2) * cnbx;
                            uint2 qa = make_uint2(0u, 0u), qb = make_uint2(0u, 0u);
                            if ((unsigned)bxa < (unsigned)cnbx) {
                                const int rb = rowb + bxa;
                                const uint4 rf = ldg(S.flagrec + dr.x + 4u * (uint32_t)(rb >> 5));
                                const uint32_t rbit = 1u << (rb & 31);
                                if (rf.x & rbit) qa = bise_row4(S.pay + dr.y, ((rf.y + popc(rf.x & (rbit - 1u))) << 4) + j0, dr.w, lut);
                            }
                            if ((o || fx) && (unsigned)(bxa + 1) < (unsigned)cnbx) {
                                const int rb = rowb + bxa + 1;
                                const uint4 rf = ldg(S.flagrec + dr.x + 4u * (uint32_t)(rb >> 5));
                                const uint32_t rbit = 1u << (rb & 31);
                                if (rf.x & rbit) qb = bise_row4(S.pay + dr.y, ((rf.y + popc(rf.x & (rbit - 1u))) << 4) + j0, dr.w, lut);
                            }
                            // samples o .. o+4 of the 8-sample string qa | qb
                            uint32_t w0 = qa.x, w1 = qa.y, w2 = qb.x, w3 = qb.y;
                            if (o & 2) { w0 = w1; w1 = w2; w2 = w3; w3 = 0u; }
                            const uint32_t sh = (uint32_t)(o & 1) << 4;
                            const uint32_t q01 = __funnelshift_r(w0, w1, sh), q23 = __funnelshift_r(w1, w2, sh), q45 = __funnelshift_r(w2, w3, sh);
                            const int q0 = (int)(int16_t)(q01 & 0xFFFFu), q1 = (int)q01 >> 16, q2 = (int)(int16_t)(q23 & 0xFFFFu), q3 = (int)q23 >> 16;
                            const int q4 = (int)(int16_t)(q45 & 0xFFFFu);
                            h0 += q0 + (fx ? q1 : 0); h1 += q1 + (fx ? q2 : 0); h2 += q2 + (fx ? q3 : 0); h3 += q3 + (fx ? q4 : 0);
                        }
                        const int k = fx + fy;  // log2 of the number of samples; rounding term n / 2 = 0, 1, 2 = k
                        const int q0 = (h0 + k) >> k, q1 = (h1 + k) >> k, q2 = (h2 + k) >> k, q3 = (h3 + k) >> k;
                        if (md) { e0 -= q0; e1 -= q1; e2 -= q2; e3 -= q3; }
                        else { e0 += q0; e1 += q1; e2 += q2; e3 += q3; }
                    }
                }
                if (!csh) { a[c][0] += e0; a[c][1] += e1; a[c][2] += e2; a[c][3] += e3; }
                else {  // chroma samples (s0 >> 1) and (s0 >> 1) + 1: elements 0, 1 or 2, 3 of the decoded row
                    const bool hi = ((s0 >> 1) & 2) != 0;
                    const int ea = hi ? e2 : e0, eb = hi ? e3 : e1;
                    a[c][0] += ea; a[c][1] += ea; a[c][2] += eb; a[c][3] += eb;
                }
            }
        }
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int acc[3] = {a[0][i], a[1][i], a[2][i]};
            rgb[i] = ycocg_to_rgb8(acc);
        }
    } else {
        atomicAdd(oob, 4ull);
    }
    uint8_t *o = kBlocks ? out + 12 * (size_t)g : out + 3 * (((size_t)view * (size_t)S.Ht + (size_t)t) * (size_t)S.Ws + (size_t)s0);
    if (out_aligned) {
        uint32_t *o32 = reinterpret_cast<uint32_t *>(o);
        o32[0] = rgb[0] | (rgb[1] << 24);
        o32[1] = (rgb[1] >> 8) | (rgb[2] << 16);
        o32[2] = (rgb[2] >> 16) | (rgb[3] << 8);
    } else {
#pragma unroll
        for (int p = 0; p < 4; ++p) {
            o[3 * p + 0] = (uint8_t)(rgb[p] & 0xFF);
            o[3 * p + 1] = (uint8_t)((rgb[p] >> 8) & 0xFF);
            o[3 * p + 2] = (uint8_t)((rgb[p] >> 16) & 0xFF);
        }
    }
}

}  // namespace

cudaError_t launch_decode_rows(const DevStream &S, const int32_t *d_views, int64_t n_views, uint8_t *d_out, unsigned long long *d_oob,
                               cudaStream_t st, int *n_launches)
{
    if (n_views == 0) return cudaSuccess;
    if (S.B != 4) return cudaErrorInvalidValue;
    const long long n_seg = (long long)n_views * S.nbx * S.Ht;
    const long long blocks = (n_seg + kNT - 1) / kNT;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidValue;
    const int aligned = ((reinterpret_cast<uintptr_t>(d_out) & 3u) == 0) ? 1 : 0;
    if (S.cs && S.sp) decode_rows_kernel<false, true, true><<<(unsigned)blocks, kNT, 0, st>>>(S, reinterpret_cast<const int2 *>(d_views), n_seg, d_out, d_oob, aligned);
    else if (S.cs) decode_rows_kernel<false, false, true><<<(unsigned)blocks, kNT, 0, st>>>(S, reinterpret_cast<const int2 *>(d_views), n_seg, d_out, d_oob, aligned);
    else if (S.sp) decode_rows_kernel<false, true><<<(unsigned)blocks, kNT, 0, st>>>(S, reinterpret_cast<const int2 *>(d_views), n_seg, d_out, d_oob, aligned);
    else decode_rows_kernel<false><<<(unsigned)blocks, kNT, 0, st>>>(S, reinterpret_cast<const int2 *>(d_views), n_seg, d_out, d_oob, aligned);
    if (n_launches) *n_launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_decode_block_rows(const DevStream &S, const int32_t *d_blocks, int64_t n_blocks, uint8_t *d_out, unsigned long long *d_oob,
                                     cudaStream_t st, int *n_launches)
{
    if (n_blocks == 0) return cudaSuccess;
    if (S.B != 4) return cudaErrorInvalidValue;
    const long long n_seg = (long long)n_blocks * 4;
    const long long blocks = (n_seg + kNT - 1) / kNT;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidValue;
    const int aligned = ((reinterpret_cast<uintptr_t>(d_out) & 3u) == 0) ? 1 : 0;
    if (S.cs && S.sp) decode_rows_kernel<true, true, true><<<(unsigned)blocks, kNT, 0, st>>>(S, reinterpret_cast<const int2 *>(d_blocks), n_seg, d_out, d_oob, aligned);
    else if (S.cs) decode_rows_kernel<true, false, true><<<(unsigned)blocks, kNT, 0, st>>>(S, reinterpret_cast<const int2 *>(d_blocks), n_seg, d_out, d_oob, aligned);
    else if (S.sp) decode_rows_kernel<true, true><<<(unsigned)blocks, kNT, 0, st>>>(S, reinterpret_cast<const int2 *>(d_blocks), n_seg, d_out, d_oob, aligned);
    else decode_rows_kernel<true><<<(unsigned)blocks, kNT, 0, st>>>(S, reinterpret_cast<const int2 *>(d_blocks), n_seg, d_out, d_oob, aligned);
    if (n_launches) *n_launches += 1;
    return cudaGetLastError();
}

}  // namespace hmlfc
