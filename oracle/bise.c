/* HMLFC oracle (test infrastructure) -- Bounded Integer Sequence Encoding.
 *
 * PAPER.md:272 (section 4.6): BISE encodes "a sequence of integer values within a fixed range
 * [0, N-1] and allows for fast random access decoding in constant time"; plain bit strings
 * are "only optimal when N is a power of two"; otherwise BISE is "close to the information
 * theoretic bounds".  The paper delegates the details to ASTC; reading R15:
 *
 *   layout = cheapest bits/value of
 *     plain : b = ceil(log2 N) bits per value
 *     trit  : smallest m with 3*2^m >= N : groups of 5 values in 8 + 5m bits
 *     quint : smallest m with 5*2^m >= N : groups of 3 values in 7 + 3m bits
 *   (ties: plain, then trit, then quint).  value = digit * 2^m + low.
 *   Bit string is LSB-first: bit j lives in byte j/8 at position j%8.
 *   trit group g (values 5g..5g+4) starts at bit g*(8+5m): 8-bit T = sum t_k 3^k, then the
 *   five m-bit low fields in order.  quint group g (values 3g..3g+2) starts at g*(7+3m):
 *   7-bit Q = sum q_k 5^k, then three m-bit low fields.  Trailing partial groups are
 *   padded with zero values.  Value i is addressable from i alone (fixed stride).
 */
#include "hmlfc_oracle.h"

static int ceil_log2_u32(uint32_t n)
{
    int b = 0;
    while (((uint64_t)1 << b) < (uint64_t)n) ++b;
    return b;
}

void orc_bise_choose(uint32_t N, int32_t *layout, int32_t *m)
{
    if (N <= 1) { *layout = ORC_BISE_PLAIN; *m = 0; return; }
    int b = ceil_log2_u32(N);
    int mt = 0;
    while ((uint64_t)3 << mt < (uint64_t)N) ++mt;
    int mq = 0;
    while ((uint64_t)5 << mq < (uint64_t)N) ++mq;
    /* bits per value scaled by 15: plain 15 b ; trit (8 + 5 m)/5 * 15 = 24 + 15 m ; quint (7 + 3 m)/3 * 15 = 35 + 15 m */
    int cost_plain = 15 * b;
    int cost_trit = 24 + 15 * mt;
    int cost_quint = 35 + 15 * mq;
    *layout = ORC_BISE_PLAIN;
    *m = b;
    int best = cost_plain;
    if (cost_trit < best) { best = cost_trit; *layout = ORC_BISE_TRIT; *m = mt; }
    if (cost_quint < best) { best = cost_quint; *layout = ORC_BISE_QUINT; *m = mq; }
}

uint64_t orc_bise_nbits(uint32_t N, uint64_t count)
{
    int32_t layout, m;
    orc_bise_choose(N, &layout, &m);
    if (layout == ORC_BISE_PLAIN) return count * (uint64_t)m;
    if (layout == ORC_BISE_TRIT) return ((count + 4) / 5) * (uint64_t)(8 + 5 * m);
    return ((count + 2) / 3) * (uint64_t)(7 + 3 * m);
}

static void put_bits(uint8_t *bits, uint64_t pos, int n, uint32_t v)
{
    for (int j = 0; j < n; ++j) {
        uint64_t p = pos + (uint64_t)j;
        if ((v >> j) & 1u) bits[p >> 3] |= (uint8_t)(1u << (p & 7));
    }
}

static uint32_t get_bits(const uint8_t *bits, uint64_t pos, int n)
{
    uint32_t v = 0;
    for (int j = 0; j < n; ++j) {
        uint64_t p = pos + (uint64_t)j;
        v |= (uint32_t)((bits[p >> 3] >> (p & 7)) & 1u) << j;
    }
    return v;
}

int orc_bise_encode(const uint32_t *values, uint64_t count, uint32_t N, uint8_t *bits)
{
    int32_t layout, m;
    orc_bise_choose(N, &layout, &m);
    for (uint64_t i = 0; i < count; ++i)
        if (values[i] >= (N ? N : 1)) return ORC_E_PARAM;
    if (layout == ORC_BISE_PLAIN) {
        for (uint64_t i = 0; i < count; ++i) put_bits(bits, i * (uint64_t)m, m, values[i]);
        return ORC_OK;
    }
    int G = (layout == ORC_BISE_TRIT) ? 5 : 3;       /* values per group */
    int base = (layout == ORC_BISE_TRIT) ? 3 : 5;    /* digit radix      */
    int hb = (layout == ORC_BISE_TRIT) ? 8 : 7;      /* bits of the packed digit word */
    uint64_t stride = (uint64_t)(hb + G * m);
    uint64_t ngroups = (count + (uint64_t)G - 1) / (uint64_t)G;
    for (uint64_t g = 0; g < ngroups; ++g) {
        uint32_t word = 0, pw = 1;
        for (int k = 0; k < G; ++k) {
            uint64_t i = g * (uint64_t)G + (uint64_t)k;
            uint32_t v = (i < count) ? values[i] : 0u;
            uint32_t digit = v >> m;
            uint32_t low = v & (((uint32_t)1 << m) - 1u);
            word += digit * pw;
            pw *= (uint32_t)base;
            put_bits(bits, g * stride + (uint64_t)hb + (uint64_t)(k * m), m, low);
        }
        put_bits(bits, g * stride, hb, word);
    }
    return ORC_OK;
}

uint32_t orc_bise_decode_at(const uint8_t *bits, uint32_t N, uint64_t i)
{
    int32_t layout, m;
    orc_bise_choose(N, &layout, &m);
    if (layout == ORC_BISE_PLAIN) return get_bits(bits, i * (uint64_t)m, m);
    int G = (layout == ORC_BISE_TRIT) ? 5 : 3;
    uint32_t base = (layout == ORC_BISE_TRIT) ? 3u : 5u;
    int hb = (layout == ORC_BISE_TRIT) ? 8 : 7;
    uint64_t stride = (uint64_t)(hb + G * m);
    uint64_t g = i / (uint64_t)G;
    int k = (int)(i % (uint64_t)G);
    uint32_t word = get_bits(bits, g * stride, hb);
    for (int j = 0; j < k; ++j) word /= base;
    uint32_t digit = word % base;
    uint32_t low = get_bits(bits, g * stride + (uint64_t)hb + (uint64_t)(k * m), m);
    return (digit << m) | low;
}

/* Sequential decode: walks a running bit cursor group by group -- deliberately a different
 * routine from decode_at (no i -> address arithmetic), so that the two pin each other. */
void orc_bise_decode_seq(const uint8_t *bits, uint32_t N, uint64_t count, uint32_t *out)
{
    int32_t layout, m;
    orc_bise_choose(N, &layout, &m);
    uint64_t cur = 0;
    if (layout == ORC_BISE_PLAIN) {
        for (uint64_t i = 0; i < count; ++i) { out[i] = get_bits(bits, cur, m); cur += (uint64_t)m; }
        return;
    }
    int G = (layout == ORC_BISE_TRIT) ? 5 : 3;
    uint32_t base = (layout == ORC_BISE_TRIT) ? 3u : 5u;
    int hb = (layout == ORC_BISE_TRIT) ? 8 : 7;
    uint64_t i = 0;
    while (i < count) {
        uint32_t word = get_bits(bits, cur, hb);
        cur += (uint64_t)hb;
        for (int k = 0; k < G; ++k) {
            uint32_t digit = word % base;
            word /= base;
            uint32_t low = get_bits(bits, cur, m);
            cur += (uint64_t)m;
            if (i < count) out[i] = (digit << m) | low;
            ++i;
        }
    }
}
