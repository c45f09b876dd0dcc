// Device-side data layout and per-sample decode of the HMLFC representation (sm_100a).
//
// What is computed: PAPER.md:289-293 (section 4.8.1, decoding procedure) and :309 (random access):
//   sample(u,v,s,t,c) = topRKV_c[v>>h][u>>h][t][s] + sum_{L<h} SRV_L[(u>>L, v>>L)](s,t)
//   SRV_L[p](s,t)     = stored_p(s,t)                                   p reference plane
//                     = stored_p(s,t) +- stored_r(s+dx, t+dy)           p predictive, block predicted
// with r the cluster's reference plane, (mode,dx,dy) the block's BISE-coded motion record
// (PAPER.md:276), stored_*(.) = 0 where the block is insignificant or outside the
// image, then inverse YCoCg-R and clamp.  Readings: DESIGN.md R7-R19.
//
// HBM layout (built by hmlfc_load):
//   pc[]       one 16-byte descriptor per SRV plane-channel: {flag record base, payload word base,
//              MV word base, offset:16 | layout:2 | m:4 | predictive:1}; the three channels of a
//              plane are adjacent (48 bytes)
//   flagrec[]  one 16-byte record per 32 blocks of a plane-channel: {res bits, res rank before,
//              pred bits, pred rank before} -- flag test and rank come from ONE 128-bit load.  The records of
//              the three channels of a (plane, group) share one 64-byte slot {Y, Co, Cg, spare}: a random
//              sample touches one HBM access granule per level instead of three (profiles/r01_cfg5.md)
//   pay[], mv[] bit-packed BISE strings as streamed (LSB-first 32-bit words), addressed in O(1)
//   rkv[]      top-level RKVs as short4 {Y, Co, Cg, 0} per sample: one 64-bit load per sample
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#define HMLFC_DEV __device__ __forceinline__

namespace hmlfc {

constexpr int kMaxLevels = 8;

struct LevelDesc {
    int32_t UL, VL;    // planes per row / rows of level L
    uint32_t pc_base;  // index of the level's first plane-channel descriptor
    uint32_t _pad;
};

struct DevStream {
    int32_t U, V, Ws, Ht, h, B, logB, W;
    int32_t nbx, nby, nblk, fgroups;  // blocks per row / column / plane; 32-block groups per plane-channel
    int32_t UH, VH;                   // top-level RKV grid
    // chroma subsampling (R18): cs = 1: the Co / Cg planes of every level are Ws/2 x Ht/2 (sample (s >> 1, t >> 1));
    // their block grid is nbx_c x nby_c.  cs = 0: the chroma fields repeat the luma ones.  (The top-level RKVs are stored at full
    // resolution on the device either way: hmlfc_load replicates subsampled chroma.)
    int32_t cs, nbx_c, nby_c, nblk_c;
    // half-pel motion compensation (R28): sp = 1: motion offsets count half pixels; mv_off = the largest offset
    // (W, or 2W), nd = 2 mv_off + 1
    int32_t sp, mv_off;
    uint32_t nd, nd2, nd_magic;       // 2W+1, (2W+1)^2, ceil(2^32 / nd)
    uint32_t mv_layout, mv_m;         // BISE layout of the motion records, N = 2 (2W+1)^2
    int32_t lmin;                     // progressive decoding (R26): levels below lmin are not summed; 0 = full quality
    LevelDesc lev[kMaxLevels];
    const uint4 *pc;
    const uint4 *flagrec;
    const uint32_t *pay;
    const uint32_t *mv;
    const short4 *rkv;
    // block records (full-resolution chroma only; null otherwise): the stored values and motion records of a plane once more, regrouped
    // per BLOCK so that what one sample needs from a plane lies in one or two sectors -- see brec_locate below
    const uint4 *pb;       // per plane {first word of the plane in brec[], wY | wCo << 8 | wCg << 16 | wMV << 24, offY | offCo << 16, offCg}
    const uint4 *bslot;    // two per (plane, 32-block group): the group's slot
    const uint32_t *brec;
    uint32_t mv_w;         // bits of a motion record as a plain binary field
    float uv_origin[2], uv_step[2], st_origin[2], st_step[2], z_st;
    float uv_inv[2], st_inv[2];  // 1 / step where that is exact (step a power of two), see pow2_mask
    uint32_t pow2_mask;          // bit 0..3: uv_step[0], uv_step[1], st_step[0], st_step[1] is a power of two
    uint32_t l2_resident;        // the device form of the stream fits the L2 with room to spare and is sparse (kernel choice of hmlfc_decode)
    uint8_t bg[4];
};

// ---------------------------------------------------------------- small helpers
template <typename T>
HMLFC_DEV T ldg(const T *p)
{
    return __ldg(p);
}

// 256-bit load (LDG.E.ENL2.256, sm_100a): two adjacent 16-byte records of a 32-byte aligned pair in one request
HMLFC_DEV void ldg256(const uint4 *__restrict__ p, uint4 &a, uint4 &b)
{
    asm volatile("ld.global.nc.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(a.x), "=r"(a.y), "=r"(a.z), "=r"(a.w), "=r"(b.x), "=r"(b.y), "=r"(b.z), "=r"(b.w) : "l"(p));
}

// the same through the L2 only (ld.global.cg): a random sector that the L1 would not see again anyway
HMLFC_DEV void ldcg256(const uint4 *__restrict__ p, uint4 &a, uint4 &b)
{
    asm volatile("ld.global.cg.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(a.x), "=r"(a.y), "=r"(a.z), "=r"(a.w), "=r"(b.x), "=r"(b.y), "=r"(b.z), "=r"(b.w) : "l"(p));
}

HMLFC_DEV uint32_t funnel_r(uint32_t lo, uint32_t hi, uint32_t sh)
{
    return __funnelshift_r(lo, hi, sh);
}

HMLFC_DEV uint32_t popc(uint32_t x)
{
    return (uint32_t)__popc(x);
}

HMLFC_DEV uint32_t umulhi(uint32_t a, uint32_t b)
{
    return __umulhi(a, b);
}

// index of the flag record of plane-channel k (= 3 * plane + channel), 32-block group g; equals pc[k].x + 4 g
HMLFC_DEV size_t flag_index(const DevStream &S, uint32_t k, uint32_t g)
{
    const uint32_t p = umulhi(k, 0xAAAAAAABu) >> 1;  // k / 3
    return ((size_t)p * (size_t)S.fgroups + (size_t)g) * 4u + (size_t)(k - 3u * p);
}

// descriptor fields
HMLFC_DEV int pc_offset(uint32_t w) { return (int)(int16_t)(w & 0xFFFFu); }
HMLFC_DEV uint32_t pc_layout(uint32_t w) { return (w >> 16) & 3u; }
HMLFC_DEV uint32_t pc_m(uint32_t w) { return (w >> 18) & 15u; }
HMLFC_DEV uint32_t pc_is_pred(uint32_t w) { return (w >> 22) & 1u; }

// ---------------------------------------------------------------- BISE decode_at
// Bit string = LSB-first 32-bit words.  plain: value i at bit i*m.  trit: group g = i/5 at bit
// g*(8+5m): 8-bit T = sum t_k 3^k then five m-bit fields.  quint: group g = i/3 at bit g*(7+3m):
// 7-bit Q = sum q_k 5^k then three m-bit fields.  value = digit * 2^m + low.  (R15)
HMLFC_DEV uint32_t bise_decode_at(const uint32_t *__restrict__ w, uint32_t i, uint32_t layout, uint32_t m)
{
    if (layout == 0u) {
        uint32_t bit = i * m;
        uint32_t idx = bit >> 5;
        uint32_t v = funnel_r(ldg(w + idx), ldg(w + idx + 1), bit & 31u);
        return v & ((1u << m) - 1u);
    }
    uint32_t g, k, gb, hb;
    if (layout == 1u) { g = i / 5u; k = i - 5u * g; hb = 8u; gb = g * (8u + 5u * m); }
    else              { g = i / 3u; k = i - 3u * g; hb = 7u; gb = g * (7u + 3u * m); }
    uint32_t idx = gb >> 5, sh = gb & 31u;
    // three words cover the digit word and every field that ends within 96 bits of the first word: all payload groups
    // (N <= 4096: at most 8 + 5*11 = 63 bits from bit sh <= 31).  Motion records of wide windows have longer groups (W = 51..54:
    // trit m = 13, 73 bits); a field that ends beyond the third word is read with its own two-word fetch.
    uint32_t w0 = ldg(w + idx), w1 = ldg(w + idx + 1), w2 = ldg(w + idx + 2);
    uint32_t head = funnel_r(w0, w1, sh) & ((1u << hb) - 1u);
    uint32_t p = sh + hb + k * m;
    uint32_t a = p < 32u ? w0 : (p < 64u ? w1 : w2);
    uint32_t b = p < 32u ? w1 : (p < 64u ? w2 : 0u);
    if (p + m > 96u) {
        const uint32_t fb = gb + hb + k * m;
        a = ldg(w + (fb >> 5));
        b = ldg(w + (fb >> 5) + 1);
    }
    uint32_t low = funnel_r(a, b, p & 31u) & ((1u << m) - 1u);
    uint32_t digit;
    if (layout == 1u) {
        // floor(T / 3^k) for T < 256 by multiply-shift, then mod 3
        uint32_t mul = k == 0u ? 65536u : k == 1u ? 21846u : k == 2u ? 7282u : k == 3u ? 2428u : 810u;
        uint32_t x = (head * mul) >> 16;
        digit = x - 3u * ((x * 171u) >> 9);
    } else {
        uint32_t mul = k == 0u ? 65536u : k == 1u ? 13108u : 2622u;
        uint32_t x = (head * mul) >> 16;
        digit = x - 5u * ((x * 205u) >> 10);
    }
    return (digit << m) | low;
}

// stored value of a plane-channel at pixel (x,y) given its descriptor and the block's flag record
HMLFC_DEV int stored_value(const DevStream &S, uint4 d, uint4 fr, uint32_t bit, int kin)
{
    if (!(fr.x & bit)) return 0;
    uint32_t rank = fr.y + popc(fr.x & (bit - 1u));
    uint32_t i = (rank << (2 * S.logB)) + (uint32_t)kin;
    return pc_offset(d.w) + (int)bise_decode_at(S.pay + d.y, i, pc_layout(d.w), pc_m(d.w));
}

// reference-plane sample at (rx,ry): 0 outside the image (R8) or in an insignificant block
HMLFC_DEV int reference_value(const DevStream &S, uint4 d, int rx, int ry, int Wc, int Hc, int nbx)
{
    if ((unsigned)rx >= (unsigned)Wc || (unsigned)ry >= (unsigned)Hc) return 0;
    int b = (ry >> S.logB) * nbx + (rx >> S.logB);
    uint4 fr = ldg(S.flagrec + d.x + 4u * (uint32_t)(b >> 5));
    int kin = ((ry & (S.B - 1)) << S.logB) + (rx & (S.B - 1));
    return stored_value(S, d, fr, 1u << (b & 31), kin);
}

// ---------------------------------------------------------------- block records (device form, hmlfc_load)
// The serialized stream keeps one BISE string per plane-channel, so the (up to) three stored values and three motion records one
// sample needs from a plane lie in six unrelated places, behind three flag records and three descriptors.  hmlfc_load re-packs them
// per plane as plain binary fields, block after block in raster order, every block that carries anything as ONE record:
//     [motion record of Y, Co, Cg where the pred flag is set : wMV bits each]
//     [sample 0: value of Y, Co, Cg where the res flag is set : wY, wCo, wCg bits][sample 1: ...] ... [sample B^2 - 1]
// (value = code, without the channel's offset; w = bits of the channel's alphabet), and keeps one 32-byte SLOT per 32 blocks of a plane:
//     bslot = {res bits Y, Co, Cg, pred bits Y, Co, Cg, first bit of the group's first record (from the plane's start), 0}
// The record of block b starts where the group starts plus the sizes of the group's records before b: popcounts of the six words.
// One sector says whether a plane holds anything for a sample and where; one or two more hold all of it.
struct BrecPos {
    unsigned long long bit;  // first bit of the block's record in brec[]
    uint32_t res, pred;      // 3-bit masks of the block's set flags
    uint32_t stride;         // bits per sample
};

// a, b = the two halves of the slot of the block's group, bit = 1 << (block & 31), pb = the plane's record descriptor
HMLFC_DEV BrecPos brec_locate(const DevStream &S, uint4 a, uint4 b, uint32_t bit, uint4 pb)
{
    const uint32_t below = bit - 1u;
    const uint32_t wY = pb.y & 0xFFu, wCo = (pb.y >> 8) & 0xFFu, wCg = (pb.y >> 16) & 0xFFu, wMV = pb.y >> 24;
    BrecPos r;
    r.res = ((a.x & bit) ? 1u : 0u) | ((a.y & bit) ? 2u : 0u) | ((a.z & bit) ? 4u : 0u);
    r.pred = ((a.w & bit) ? 1u : 0u) | ((b.x & bit) ? 2u : 0u) | ((b.y & bit) ? 4u : 0u);
    r.stride = ((r.res & 1u) ? wY : 0u) + ((r.res & 2u) ? wCo : 0u) + ((r.res & 4u) ? wCg : 0u);
    const uint32_t before = ((popc(a.x & below) * wY + popc(a.y & below) * wCo + popc(a.z & below) * wCg) << (2 * S.logB)) +
                            (popc(a.w & below) + popc(b.x & below) + popc(b.y & below)) * wMV;
    r.bit = (unsigned long long)pb.x * 32ull + (unsigned long long)b.z + (unsigned long long)before;
    return r;
}

// bit offset (from the record's start) of the motion record of channel c / of sample kin's first value / of channel c within a sample
HMLFC_DEV uint32_t brec_mv_offset(const BrecPos &r, uint4 pb, int c) { return popc(r.pred & ((1u << c) - 1u)) * (pb.y >> 24); }
HMLFC_DEV uint32_t brec_sample_offset(const BrecPos &r, uint4 pb, uint32_t kin) { return popc(r.pred) * (pb.y >> 24) + kin * r.stride; }
HMLFC_DEV uint32_t brec_channel_offset(const BrecPos &r, uint4 pb, int c)
{
    uint32_t before = 0u;
    if (c > 0 && (r.res & 1u)) before += pb.y & 0xFFu;
    if (c > 1 && (r.res & 2u)) before += (pb.y >> 8) & 0xFFu;
    return before;
}
HMLFC_DEV int brec_offset_of(uint4 pb, int c) { return (int)(int16_t)(c == 0 ? pb.z & 0xFFFFu : c == 1 ? pb.z >> 16 : pb.w & 0xFFFFu); }

// 96-bit window of brec[] from the word that holds bit `bit`: an aligned 64-bit load, the next pair only when `span` bits from `bit`
// leave the first (at most 96 - 31 = 65 bits are needed by any caller)
struct BrecWindow { uint32_t w0, w1, w2; };
template <bool kCg = false>
HMLFC_DEV BrecWindow brec_window(const uint32_t *__restrict__ brec, unsigned long long bit, uint32_t span)
{
    const unsigned long long wi = bit >> 5;
    const uint32_t odd = (uint32_t)wi & 1u, sh = (uint32_t)bit & 31u;
    const uint2 *p2 = reinterpret_cast<const uint2 *>(brec + (wi & ~1ull));
    const uint2 A = kCg ? __ldcg(p2) : __ldg(p2);
    uint2 B = make_uint2(0u, 0u);
    if (odd * 32u + sh + span > 64u) B = kCg ? __ldcg(p2 + 1) : __ldg(p2 + 1);
    BrecWindow r;
    r.w0 = odd ? A.y : A.x; r.w1 = odd ? B.x : A.y; r.w2 = odd ? B.y : B.x;
    return r;
}
// the w-bit field (w <= 16) at bit `pos` (< 80) of the window
HMLFC_DEV uint32_t brec_window_field(const BrecWindow &q, uint32_t pos, uint32_t w)
{
    const uint32_t lo = pos < 32u ? q.w0 : (pos < 64u ? q.w1 : q.w2), hi = pos < 32u ? q.w1 : (pos < 64u ? q.w2 : 0u);
    return funnel_r(lo, hi, pos & 31u) & ((1u << w) - 1u);
}

// reference value at the half-pel position (x2 / 2, y2 / 2) (R28): the mean of the 1, 2 or 4 stored reference samples around
// it, rounded half up (arithmetic shifts = floor), each sample 0 outside the image or in an insignificant block
HMLFC_DEV int reference_halfpel(const DevStream &S, uint4 d, int x2, int y2, int Wc, int Hc, int nbx)
{
    const int x0 = x2 >> 1, y0 = y2 >> 1, fx = x2 & 1, fy = y2 & 1;
    int s = reference_value(S, d, x0, y0, Wc, Hc, nbx);
    if (fx) s += reference_value(S, d, x0 + 1, y0, Wc, Hc, nbx);
    if (fy) {
        s += reference_value(S, d, x0, y0 + 1, Wc, Hc, nbx);
        if (fx) s += reference_value(S, d, x0 + 1, y0 + 1, Wc, Hc, nbx);
    }
    const int k = fx + fy;  // log2 of the number of samples; the rounding term n / 2 = 0, 1, 2 = k
    return (s + k) >> k;
}

// motion record r = mode*nd^2 + (dy+off)*nd + (dx+off), off = mv_off  (R16, R28)
HMLFC_DEV void mv_unpack(const DevStream &S, uint32_t r, int &mode, int &dx, int &dy)
{
    mode = r >= S.nd2;
    uint32_t rem = r - (mode ? S.nd2 : 0u);
    uint32_t q = umulhi(rem, S.nd_magic);  // exact floor(rem / nd) for rem < 2^16
    dy = (int)q - S.mv_off;
    dx = (int)(rem - q * S.nd) - S.mv_off;
}

// (Y, Co, Cg) of light-field sample (u,v,s=x,t=y); coordinates must be in range
HMLFC_DEV void decode_ycocg(const DevStream &S, int u, int v, int x, int y, int acc[3])
{
    const int h = S.h;
    size_t ri = ((size_t)((v >> h) * S.UH + (u >> h)) * (size_t)S.Ht + (size_t)y) * (size_t)S.Ws + (size_t)x;
    short4 r = ldg(S.rkv + ri);
    acc[0] = r.x; acc[1] = r.y; acc[2] = r.z;
    // block, flag bit and position in the block for luma [0] and for chroma [1] (the chroma sample of (x,y) is (x >> cs, y >> cs), R18)
    const int xc = x >> S.cs, yc = y >> S.cs;
    const int b2[2] = {(y >> S.logB) * S.nbx + (x >> S.logB), (yc >> S.logB) * S.nbx_c + (xc >> S.logB)};
    const int kin2[2] = {((y & (S.B - 1)) << S.logB) + (x & (S.B - 1)), ((yc & (S.B - 1)) << S.logB) + (xc & (S.B - 1))};
#pragma unroll 1
    for (int L = S.lmin; L < h; ++L) {
        const int pu = u >> L, pv = v >> L;
        const LevelDesc lv = S.lev[L];
        const uint32_t base = lv.pc_base + (uint32_t)(pv * lv.UL + pu) * 3u;
        const uint32_t rbase = lv.pc_base + (uint32_t)((pv & ~1) * lv.UL + (pu & ~1)) * 3u;
        const bool predictive = ((pu | pv) & 1) != 0;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const int b = b2[c > 0], kin = kin2[c > 0];
            const uint32_t bit = 1u << (b & 31), fg = (uint32_t)(b >> 5);
            uint4 d = ldg(S.pc + base + c);
            // the flag record's index follows from the plane-channel index (= d.x + 4 fg): both loads issue at once
            uint4 fr = ldg(S.flagrec + flag_index(S, base + (uint32_t)c, fg));
            int e = stored_value(S, d, fr, bit, kin);
            if (predictive && (fr.z & bit)) {
                uint32_t mi = fr.w + popc(fr.z & (bit - 1u));
                uint32_t rec = bise_decode_at(S.mv + d.z, mi, S.mv_layout, S.mv_m);
                int mode, dx, dy;
                mv_unpack(S, rec, mode, dx, dy);
                const uint4 rd = ldg(S.pc + rbase + c);
                const int px = c > 0 ? xc : x, py = c > 0 ? yc : y;
                const int Wc = c > 0 ? (S.Ws >> S.cs) : S.Ws, Hc = c > 0 ? (S.Ht >> S.cs) : S.Ht, nbxc = c > 0 ? S.nbx_c : S.nbx;
                const int q = S.sp ? reference_halfpel(S, rd, 2 * px + dx, 2 * py + dy, Wc, Hc, nbxc)
                                   : reference_value(S, rd, px + dx, py + dy, Wc, Hc, nbxc);
                e += mode ? -q : q;  // R10: subtractive P = e + R, additive P = e - R
            }
            acc[c] += e;
        }
    }
}

// inverse YCoCg-R (arithmetic shifts = floor) and clamp to [0,255]; returns R | G<<8 | B<<16
HMLFC_DEV uint32_t ycocg_to_rgb8(const int acc[3])
{
    int t = acc[0] - (acc[2] >> 1);
    int G = acc[2] + t;
    int Bl = t - (acc[1] >> 1);
    int R = Bl + acc[1];
    R = min(max(R, 0), 255);
    G = min(max(G, 0), 255);
    Bl = min(max(Bl, 0), 255);
    return (uint32_t)R | ((uint32_t)G << 8) | ((uint32_t)Bl << 16);
}

HMLFC_DEV uint32_t decode_rgb8(const DevStream &S, int u, int v, int x, int y)
{
    int acc[3];
    decode_ycocg(S, u, v, x, y, acc);
    return ycocg_to_rgb8(acc);
}

// ---------------------------------------------------------------- ray set-up
// Strict IEEE fp32, fixed operation order, no FMA contraction: __fmul_rn/__fadd_rn/__fdiv_rn are
// never fused by the compiler, so hit/miss and floor() agree bit for bit with the oracle.
struct Camera {
    float eye[3], right[3], down[3], fwd[3];
    float tan_half_x, tan_half_y;
    float _pad[2];
};

struct Ray {
    float u, v, s, t;
    bool hit;
};

#define HMLFC_MUL(a, b) __fmul_rn((a), (b))
#define HMLFC_ADD(a, b) __fadd_rn((a), (b))
#define HMLFC_SUB(a, b) __fsub_rn((a), (b))
#define HMLFC_DIV(a, b) __fdiv_rn((a), (b))

// x / step.  When step is a power of two, x * (1/step) is the same correctly rounded real number, so
// the multiplication is bit-identical to the IEEE division the definition asks for.
HMLFC_DEV float div_step(float x, float step, float inv, bool pow2) { return pow2 ? HMLFC_MUL(x, inv) : HMLFC_DIV(x, step); }

// screen coordinate of pixel column / row i of an n-pixel-wide view: ((2 (i + 0.5)) / n - 1) tan_half
HMLFC_DEV float ray_screen(float tan_half, int n, int i)
{
    return HMLFC_MUL(HMLFC_SUB(HMLFC_DIV(HMLFC_MUL(2.0f, HMLFC_ADD((float)i, 0.5f)), (float)n), 1.0f), tan_half);
}

HMLFC_DEV Ray ray_from_screen(const DevStream &S, const Camera &cam, float px, float py);

HMLFC_DEV Ray ray_setup(const DevStream &S, const Camera &cam, int W, int H, int i, int j)
{
    return ray_from_screen(S, cam, ray_screen(cam.tan_half_x, W, i), ray_screen(cam.tan_half_y, H, j));
}

// kAllPow2: all four steps are powers of two (pow2_mask == 15): the divisions by the steps are multiplications, without the test
template <bool kAllPow2>
HMLFC_DEV Ray ray_from_screen_t(const DevStream &S, const Camera &cam, float px, float py)
{
    Ray r;
    r.hit = false;
    r.u = r.v = r.s = r.t = 0.0f;
    float Dx = HMLFC_ADD(HMLFC_ADD(cam.fwd[0], HMLFC_MUL(px, cam.right[0])), HMLFC_MUL(py, cam.down[0]));
    float Dy = HMLFC_ADD(HMLFC_ADD(cam.fwd[1], HMLFC_MUL(px, cam.right[1])), HMLFC_MUL(py, cam.down[1]));
    float Dz = HMLFC_ADD(HMLFC_ADD(cam.fwd[2], HMLFC_MUL(px, cam.right[2])), HMLFC_MUL(py, cam.down[2]));
    if (!(Dz > 0.0f)) return r;
    float l0 = HMLFC_DIV(HMLFC_SUB(0.0f, cam.eye[2]), Dz);
    float l1 = HMLFC_DIV(HMLFC_SUB(S.z_st, cam.eye[2]), Dz);
    float uw = HMLFC_ADD(cam.eye[0], HMLFC_MUL(l0, Dx));
    float vw = HMLFC_ADD(cam.eye[1], HMLFC_MUL(l0, Dy));
    float sw = HMLFC_ADD(cam.eye[0], HMLFC_MUL(l1, Dx));
    float tw = HMLFC_ADD(cam.eye[1], HMLFC_MUL(l1, Dy));
    float u = div_step(HMLFC_SUB(uw, S.uv_origin[0]), S.uv_step[0], S.uv_inv[0], kAllPow2 || (S.pow2_mask & 1u));
    float v = div_step(HMLFC_SUB(vw, S.uv_origin[1]), S.uv_step[1], S.uv_inv[1], kAllPow2 || (S.pow2_mask & 2u));
    float s = div_step(HMLFC_SUB(sw, S.st_origin[0]), S.st_step[0], S.st_inv[0], kAllPow2 || (S.pow2_mask & 4u));
    float t = div_step(HMLFC_SUB(tw, S.st_origin[1]), S.st_step[1], S.st_inv[1], kAllPow2 || (S.pow2_mask & 8u));
    if (!(u >= 0.0f && u <= (float)(S.U - 1) && v >= 0.0f && v <= (float)(S.V - 1) && s >= 0.0f &&
          s <= (float)(S.Ws - 1) && t >= 0.0f && t <= (float)(S.Ht - 1)))
        return r;
    r.hit = true;
    r.u = u; r.v = v; r.s = s; r.t = t;
    return r;
}

HMLFC_DEV Ray ray_from_screen(const DevStream &S, const Camera &cam, float px, float py)
{
    return ray_from_screen_t<false>(S, cam, px, py);
}

// 16-tap enumeration: base indices, +1 neighbours clamped to the edge, fractional weights
struct Taps {
    int u0, u1, v0, v1, s0, s1, t0, t1;
    float fu, fv, fs, ft;
};

HMLFC_DEV Taps tap_setup(const DevStream &S, const Ray &r)
{
    Taps k;
    float u0 = floorf(r.u), v0 = floorf(r.v), s0 = floorf(r.s), t0 = floorf(r.t);
    k.fu = HMLFC_SUB(r.u, u0); k.fv = HMLFC_SUB(r.v, v0); k.fs = HMLFC_SUB(r.s, s0); k.ft = HMLFC_SUB(r.t, t0);
    k.u0 = (int)u0; k.v0 = (int)v0; k.s0 = (int)s0; k.t0 = (int)t0;
    k.u1 = min(k.u0 + 1, S.U - 1);
    k.v1 = min(k.v0 + 1, S.V - 1);
    k.s1 = min(k.s0 + 1, S.Ws - 1);
    k.t1 = min(k.t0 + 1, S.Ht - 1);
    return k;
}

}  // namespace hmlfc
