// Block-row BISE decoding shared by the CTA render kernel (hmlfc_render_cta.cu) and the dense / block decode kernel
// (hmlfc_decode_rows.cu): the digit table of the packed trit / quint words, decode_at of one value (motion records) and of
// the four values of one row of a 4 x 4 block.  PAPER.md:272 (BISE), :276 (motion records); layout: DESIGN.md section 4.
#pragma once

#include "hmlfc_device.cuh"

namespace hmlfc {

// digits of the packed trit / quint words: trit T -> t0 | t1<<2 | .. | t4<<8, quint Q -> q0 | q1<<3 | q2<<6
struct DigitLut {
    uint16_t v[384];
};

constexpr DigitLut make_digit_lut()
{
    DigitLut l{};
    for (int T = 0; T < 256; ++T) {
        int x = T, p = 0;
        for (int k = 0; k < 5; ++k) { p |= (x % 3) << (2 * k); x /= 3; }
        l.v[T] = (uint16_t)p;
    }
    for (int Q = 0; Q < 128; ++Q) {
        int x = Q, p = 0;
        for (int k = 0; k < 3; ++k) { p |= (x % 5) << (3 * k); x /= 5; }
        l.v[256 + Q] = (uint16_t)p;
    }
    return l;
}

static __device__ const DigitLut g_cta_digit_lut = make_digit_lut();

// bits [pos, pos+n) of an LSB-first 32-bit word string, n <= 16
__device__ __forceinline__ uint32_t bits_at(const uint32_t *__restrict__ w, uint32_t pos, uint32_t n)
{
    const uint32_t *p = w + (pos >> 5);
    return __funnelshift_r(__ldg(p), __ldg(p + 1), pos & 31u) & ((1u << n) - 1u);
}

// BISE decode_at of one value (layout in DESIGN.md section 4) -- used for the motion records
__device__ __forceinline__ uint32_t bise_at(const uint32_t *__restrict__ w, uint32_t i, uint32_t layout, uint32_t m,
                                            const uint16_t *__restrict__ lut)
{
    if (layout == 0u) return bits_at(w, i * m, m);
    const bool trit = layout == 1u;
    const uint32_t G = trit ? 5u : 3u, hb = trit ? 8u : 7u;
    const uint32_t g = trit ? (__umulhi(i, 0xCCCCCCCDu) >> 2) : (__umulhi(i, 0xAAAAAAABu) >> 1);
    const uint32_t k = i - G * g;
    const uint32_t gb = g * (hb + G * m);
    const uint32_t head = bits_at(w, gb, hb);
    const uint32_t low = bits_at(w, gb + hb + k * m, m);
    const uint32_t dig = ((uint32_t)lut[(trit ? 0u : 256u) + head] >> (k * (trit ? 2u : 3u))) & (trit ? 3u : 7u);
    return (dig << m) | low;
}

// 64 bits of an LSB-first word string starting at bit pos
__device__ __forceinline__ uint2 window64(const uint32_t *__restrict__ w, uint32_t pos)
{
    const uint32_t *p = w + (pos >> 5);
    const uint32_t w0 = __ldg(p), w1 = __ldg(p + 1), w2 = __ldg(p + 2), sh = pos & 31u;
    return make_uint2(__funnelshift_r(w0, w1, sh), __funnelshift_r(w1, w2, sh));
}

// BISE decode of the 4 consecutive values i0 .. i0+3 (i0 a multiple of 4: one row of a 4 x 4 block) of the string
// w, plus the plane-channel's offset; returned as 4 packed int16.  The values lie in at most two consecutive
// groups (quint: 3 values per group, trit: 5; plain is read as one pseudo-group of 4 values without a digit word),
// each at most 58 bits long, so two 64-bit windows cover them.  No control flow: lanes of a warp working on
// plane-channels with different layouts do not diverge.
__device__ __forceinline__ uint2 bise_row4(const uint32_t *__restrict__ w, uint32_t i0, uint32_t dword, const uint16_t *__restrict__ lut)
{
    const uint32_t layout = pc_layout(dword), m = pc_m(dword);
    const int off = pc_offset(dword);
    const bool plain = layout == 0u, trit = layout == 1u;
    const uint32_t G = plain ? 4u : (trit ? 5u : 3u), hb = plain ? 0u : (trit ? 8u : 7u);
    const uint32_t gA = plain ? (i0 >> 2) : (trit ? (__umulhi(i0, 0xCCCCCCCDu) >> 2) : (__umulhi(i0, 0xAAAAAAABu) >> 1));
    const uint32_t kA = i0 - G * gA;
    const uint32_t gbits = hb + G * m;
    const uint32_t posA = gA * gbits;
    const uint2 A = window64(w, posA);
    uint2 Bw = make_uint2(0u, 0u);
    if (kA + 3u >= G) Bw = window64(w, posA + gbits);
    const uint32_t hmask = (1u << hb) - 1u, lmask = (1u << m) - 1u;
    const uint32_t lbase = trit ? 0u : 256u;
    const uint32_t digA = plain ? 0u : (uint32_t)lut[lbase + (A.x & hmask)];
    const uint32_t digB = plain ? 0u : (uint32_t)lut[lbase + (Bw.x & hmask)];
    const uint32_t dshift = trit ? 2u : 3u, dmask = trit ? 3u : 7u;
    uint32_t v[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        uint32_t k = kA + (uint32_t)j;
        const bool inB = k >= G;
        k = inB ? k - G : k;
        const uint32_t lo = inB ? Bw.x : A.x, hi = inB ? Bw.y : A.y, dg = inB ? digB : digA;
        const uint32_t pos = hb + k * m;
        const uint32_t bits = pos < 32u ? __funnelshift_r(lo, hi, pos) : (hi >> (pos - 32u));
        const uint32_t d = (dg >> (k * dshift)) & dmask;
        v[j] = (uint32_t)(off + (int)((d << m) | (bits & lmask))) & 0xFFFFu;
    }
    return make_uint2(v[0] | (v[1] << 16), v[2] | (v[3] << 16));
}

}  // namespace hmlfc
