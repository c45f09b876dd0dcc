// Host-side parsing of a serialized HMLFC stream into the device structure-of-arrays tables.
// Written from DESIGN.md "Stream format v1"; shares no code with the oracle's parser.
#pragma once

#include "../../include/hmlfc.h"
#include "hmlfc_device.cuh"

#include <cmath>
#include <cstring>
#include <new>
#include <vector>

namespace hmlfc {

struct HostTables {
    DevStream ds{};  // device pointers left null; hmlfc_load fills them after the upload
    hmlfc_info_t info{};
    std::vector<uint4> pc, flagrec;
    std::vector<uint4> bslot;  // block records: 32-byte slot per (plane, 32-block group)
    std::vector<uint4> pb;     // per plane: block-record descriptor (hmlfc_device.cuh, "block records"); empty for subsampled streams
    uint64_t brec_words = 0;   // 32-bit words of the block-record array (with its read slack)
    uint64_t n_flagged = 0;  // set res and pred flags of the whole stream
    std::vector<uint32_t> bits15;  // per plane-channel BISE bits/value in 1/15 bit (footprint only)
    std::vector<short4> rkv;
    uint64_t n_pc = 0, off_pay = 0, off_mv = 0, total = 0;
    uint32_t mv_bits15 = 0;
};

namespace tables_detail {

inline uint32_t rd16(const uint8_t *p) { return (uint32_t)p[0] | ((uint32_t)p[1] << 8); }
inline uint32_t rd32(const uint8_t *p) { return rd16(p) | (rd16(p + 2) << 16); }
inline uint64_t rd64(const uint8_t *p) { return (uint64_t)rd32(p) | ((uint64_t)rd32(p + 4) << 32); }
inline float rdf(const uint8_t *p) { uint32_t u = rd32(p); float f; memcpy(&f, &u, 4); return f; }

constexpr size_t kHeaderBytes = 160, kDirentBytes = 48;

// BISE layout rule (R15): cheapest bits/value of plain / trit / quint; ties in that order.
inline void bise_layout(uint32_t N, uint32_t *layout, uint32_t *m)
{
    if (N <= 1) { *layout = 0; *m = 0; return; }
    uint32_t b = 0, mt = 0, mq = 0;
    while ((1ull << b) < N) ++b;
    while ((3ull << mt) < N) ++mt;
    while ((5ull << mq) < N) ++mq;
    uint32_t cp = 15 * b, ct = 24 + 15 * mt, cq = 35 + 15 * mq;
    *layout = 0; *m = b;
    uint32_t best = cp;
    if (ct < best) { best = ct; *layout = 1; *m = mt; }
    if (cq < best) { *layout = 2; *m = mq; }
}

inline uint32_t bise_bits15(uint32_t layout, uint32_t m) { return layout == 0 ? 15 * m : layout == 1 ? 24 + 15 * m : 35 + 15 * m; }

inline uint64_t bise_nbits(uint32_t layout, uint32_t m, uint64_t count)
{
    if (layout == 0) return count * m;
    if (layout == 1) return ((count + 4) / 5) * (8 + 5 * m);
    return ((count + 2) / 3) * (7 + 3 * m);
}

inline uint32_t popcount32(uint32_t x)
{
    x = x - ((x >> 1) & 0x55555555u);
    x = (x & 0x33333333u) + ((x >> 2) & 0x33333333u);
    return (((x + (x >> 4)) & 0x0F0F0F0Fu) * 0x01010101u) >> 24;
}

}  // namespace tables_detail

// Validates the stream and fills T.  Returns HMLFC_OK or a negative HMLFC_E_* code.
inline int build_tables(const void *h_stream_bytes, size_t len, HostTables &T)
{
    using namespace tables_detail;
    const uint8_t *s = static_cast<const uint8_t *>(h_stream_bytes);
    if (len < 8) return HMLFC_E_TRUNCATED;
    if (memcmp(s, "HMLF", 4) != 0) return HMLFC_E_MAGIC;
    if (rd16(s + 4) != 1) return HMLFC_E_VERSION;
    if (len < kHeaderBytes) return HMLFC_E_TRUNCATED;

    hmlfc_info_t &I = T.info;
    I.U = (int32_t)rd32(s + 8); I.V = (int32_t)rd32(s + 12); I.Ws = (int32_t)rd32(s + 16); I.Ht = (int32_t)rd32(s + 20);
    I.height = (int32_t)rd32(s + 24); I.block = (int32_t)rd32(s + 28); I.window = (int32_t)rd32(s + 32);
    const uint32_t n_channels = rd32(s + 36);
    I.tau_ref = (int32_t)rd32(s + 40); I.tau_res = (int32_t)rd32(s + 44);
    const uint8_t colour_id = s[48], chroma = s[49], rkv_codec = s[50], subpel = s[55];
    I.background[0] = s[52]; I.background[1] = s[53]; I.background[2] = s[54];
    I.uv_origin[0] = rdf(s + 56); I.uv_origin[1] = rdf(s + 60); I.uv_step[0] = rdf(s + 64); I.uv_step[1] = rdf(s + 68);
    I.st_origin[0] = rdf(s + 72); I.st_origin[1] = rdf(s + 76); I.st_step[0] = rdf(s + 80); I.st_step[1] = rdf(s + 84);
    I.z_st = rdf(s + 88);
    const uint64_t n_pc_hdr = rd64(s + 104);
    const uint64_t off_rkv = rd64(s + 112), off_dir = rd64(s + 120), off_flags = rd64(s + 128);
    const uint64_t off_pay = rd64(s + 136), off_mv = rd64(s + 144), total = rd64(s + 152);

    if (rd16(s + 6) != kHeaderBytes) return HMLFC_E_CORRUPT;
    if (I.U < 1 || I.V < 1 || I.Ws < 1 || I.Ht < 1 || I.height < 1 || I.window < 0) return HMLFC_E_CORRUPT;
    if (n_channels != 3 || colour_id != 1 || chroma > 1 || rkv_codec != 0 || subpel > 1) return HMLFC_E_UNSUPPORTED;
    if (I.height > kMaxLevels || I.window > 64) return HMLFC_E_UNSUPPORTED;
    if (!(I.block == 2 || I.block == 4 || I.block == 8) || (I.Ws % I.block) || (I.Ht % I.block)) return HMLFC_E_UNSUPPORTED;
    // chroma subsampling (R18): Co / Cg planes at Ws/2 x Ht/2, which the blocks must tile as well
    if (chroma && ((I.Ws & 1) || (I.Ht & 1) || ((I.Ws / 2) % I.block) || ((I.Ht / 2) % I.block))) return HMLFC_E_UNSUPPORTED;
    if ((uint64_t)I.U * I.V > (1u << 24) || (uint64_t)I.Ws * I.Ht > (1u << 26)) return HMLFC_E_UNSUPPORTED;
    if (I.U > 4096 || I.V > 4096 || I.Ws > 16384 || I.Ht > 16384) return HMLFC_E_UNSUPPORTED;  // packed tap indices
    if (len < total) return HMLFC_E_TRUNCATED;

    DevStream &D = T.ds;
    D.U = I.U; D.V = I.V; D.Ws = I.Ws; D.Ht = I.Ht; D.h = I.height; D.B = I.block; D.W = I.window;
    D.logB = I.block == 2 ? 1 : I.block == 4 ? 2 : 3;
    D.nbx = I.Ws / I.block; D.nby = I.Ht / I.block; D.nblk = D.nbx * D.nby; D.fgroups = (D.nblk + 31) / 32;
    D.cs = chroma ? 1 : 0;
    D.nbx_c = (I.Ws >> D.cs) / I.block; D.nby_c = (I.Ht >> D.cs) / I.block; D.nblk_c = D.nbx_c * D.nby_c;
    // half-pel motion compensation (R28): offsets in half pixels, range [-2W, 2W]
    D.sp = subpel ? 1 : 0;
    D.mv_off = (subpel ? 2 : 1) * I.window;
    D.nd = 2u * (uint32_t)D.mv_off + 1u; D.nd2 = D.nd * D.nd;
    D.nd_magic = D.nd == 1 ? 0xFFFFFFFFu : (uint32_t)((0x100000000ull + D.nd - 1) / D.nd);
    bise_layout(2u * D.nd2, &D.mv_layout, &D.mv_m);
    D.mv_w = D.mv_m + (D.mv_layout == 0 ? 0u : D.mv_layout == 1 ? 2u : 3u);
    T.mv_bits15 = bise_bits15(D.mv_layout, D.mv_m);
    for (int i = 0; i < 2; ++i) {
        D.uv_origin[i] = I.uv_origin[i]; D.uv_step[i] = I.uv_step[i];
        D.st_origin[i] = I.st_origin[i]; D.st_step[i] = I.st_step[i];
    }
    D.z_st = I.z_st;
    D.pow2_mask = 0;
    for (int i = 0; i < 4; ++i) {  // a step whose reciprocal is exact lets the kernels multiply instead of divide
        const float step = i < 2 ? I.uv_step[i] : I.st_step[i - 2];
        int e = 0;
        const bool pow2 = std::isnormal(step) && std::frexp(step, &e) == 0.5f && std::isnormal(1.0f / step);
        (i < 2 ? D.uv_inv[i] : D.st_inv[i - 2]) = pow2 ? 1.0f / step : 0.0f;
        if (pow2) D.pow2_mask |= 1u << i;
    }
    D.bg[0] = I.background[0]; D.bg[1] = I.background[1]; D.bg[2] = I.background[2]; D.bg[3] = 0;

    // level table: the stream lists levels top-down (L = h-1 .. 0), planes row-major, channel innermost
    uint64_t n_pc = 0;
    for (int L = I.height - 1; L >= 0; --L) {
        D.lev[L].UL = (I.U + (1 << L) - 1) >> L;
        D.lev[L].VL = (I.V + (1 << L) - 1) >> L;
        D.lev[L].pc_base = (uint32_t)n_pc;
        n_pc += (uint64_t)D.lev[L].UL * D.lev[L].VL * 3;
    }
    D.UH = (I.U + (1 << I.height) - 1) >> I.height;
    D.VH = (I.V + (1 << I.height) - 1) >> I.height;
    const uint64_t npx = (uint64_t)I.Ws * I.Ht, n_top = (uint64_t)D.UH * D.VH;
    const uint64_t npx_c = (uint64_t)(I.Ws >> D.cs) * (uint64_t)(I.Ht >> D.cs);  // samples of a chroma plane
    if (n_pc != n_pc_hdr || n_pc * (uint64_t)D.fgroups > 0xFFFFFFFFull) return HMLFC_E_CORRUPT;
    if (off_rkv != kHeaderBytes || off_dir < off_rkv + n_top * (npx + 4 * npx_c) || off_flags < off_dir + n_pc * kDirentBytes ||
        off_pay < off_flags || off_mv < off_pay || total < off_mv)
        return HMLFC_E_CORRUPT;
    const uint64_t flags_len = off_pay - off_flags, pay_bits = (off_mv - off_pay) * 8, mv_bits = (total - off_mv) * 8;
    if (pay_bits / 32 > 0xFFFFFFF0ull || mv_bits / 32 > 0xFFFFFFF0ull) return HMLFC_E_UNSUPPORTED;
    T.n_pc = n_pc; T.off_pay = off_pay; T.off_mv = off_mv; T.total = total;
    I.n_plane_channels = n_pc;
    I.stream_bytes = total;

    try {
        T.pc.resize(n_pc);
        T.bits15.resize(n_pc);
        T.flagrec.assign((n_pc / 3) * (uint64_t)D.fgroups * 4, make_uint4(0u, 0u, 0u, 0u));  // 64-byte slot per (plane, group): Y, Co, Cg, bit words of Y and Co
        T.rkv.resize(n_top * npx);
        if (!D.cs && !D.sp) {
            T.pb.assign(n_pc / 3, make_uint4(0u, 0u, 0u, 0u));
            T.bslot.assign((n_pc / 3) * (uint64_t)D.fgroups * 2, make_uint4(0u, 0u, 0u, 0u));
        }
    } catch (const std::bad_alloc &) {
        return HMLFC_E_NOMEM;
    }

    // descriptors + flag/rank records
    const uint32_t BB = (uint32_t)(I.block * I.block);
    uint64_t k = 0;
    for (int L = I.height - 1; L >= 0; --L)
        for (int pv = 0; pv < D.lev[L].VL; ++pv)
            for (int pu = 0; pu < D.lev[L].UL; ++pu)
                for (int c = 0; c < 3; ++c, ++k) {
                    const uint8_t *e = s + off_dir + k * kDirentBytes;
                    const int32_t offset = (int32_t)rd32(e);
                    const uint32_t N = rd32(e + 4), n_res = rd32(e + 8), n_pred = rd32(e + 12);
                    const uint64_t foff = rd64(e + 16), pboff = rd64(e + 24), mboff = rd64(e + 32);
                    const bool is_pred = ((pu | pv) & 1) != 0;
                    const int nblk_k = c == 0 ? D.nblk : D.nblk_c, fgroups_k = (nblk_k + 31) / 32;  // the channel's own block grid
                    const uint64_t fbytes = (uint64_t)fgroups_k * 4;
                    uint32_t layout, m;
                    bise_layout(N, &layout, &m);
                    if (N < 1 || N > 4096 || offset < -32768 || offset > 32767 || e[40] != layout || e[41] != m ||
                        e[42] != (is_pred ? 1 : 0) || (pboff & 31) || (mboff & 31) || (foff & 3) ||
                        n_res > (uint32_t)nblk_k || n_pred > (uint32_t)nblk_k ||
                        // subtraction form: the 64-bit offsets are untrusted and must not wrap
                        foff > flags_len || fbytes * (is_pred ? 2 : 1) > flags_len - foff ||
                        pboff > pay_bits || bise_nbits(layout, m, (uint64_t)n_res * BB) > pay_bits - pboff ||
                        mboff > mv_bits || bise_nbits(D.mv_layout, D.mv_m, n_pred) > mv_bits - mboff || (!is_pred && n_pred != 0))
                        return HMLFC_E_CORRUPT;
                    const uint64_t frbase = (k / 3) * (uint64_t)D.fgroups * 4 + (k % 3);  // record of group g: frbase + 4 g
                    if (frbase + 4ull * (uint64_t)D.fgroups > 0xFFFFFFFFull) return HMLFC_E_UNSUPPORTED;
                    T.pc[k] = make_uint4((uint32_t)frbase, (uint32_t)(pboff / 32), (uint32_t)(mboff / 32),
                                         ((uint32_t)offset & 0xFFFFu) | (layout << 16) | (m << 18) | ((is_pred ? 1u : 0u) << 22));
                    T.bits15[k] = bise_bits15(layout, m);
                    const uint8_t *fres = s + off_flags + foff;
                    const uint8_t *fprd = fres + fbytes;
                    uint32_t rr = 0, rp = 0;
                    for (int g = 0; g < fgroups_k; ++g) {  // (a subsampled channel leaves the records of the plane's later groups empty)
                        uint32_t wr = rd32(fres + 4 * g), wp = is_pred ? rd32(fprd + 4 * g) : 0u;
                        if (g == fgroups_k - 1 && (nblk_k & 31)) {  // ignore padding bits
                            const uint32_t mask = (1u << (nblk_k & 31)) - 1u;
                            wr &= mask; wp &= mask;
                        }
                        T.flagrec[frbase + 4ull * (uint64_t)g] = make_uint4(wr, rr, wp, rp);
                        // the slot's fourth record repeats the Y and Co bit words {res Y, res Co, pred Y, pred Co}: together with the Cg
                        // record before it, ONE 32-byte sector holds all six bit words of the 32 blocks (a random sample's first look)
                        if (c < 2) {
                            uint4 &sp = T.flagrec[(k / 3) * (uint64_t)D.fgroups * 4 + 4ull * (uint64_t)g + 3];
                            if (c == 0) { sp.x = wr; sp.z = wp; } else { sp.y = wr; sp.w = wp; }
                        }
                        rr += popcount32(wr);
                        rp += popcount32(wp);
                    }
                    if (rr != n_res || rp != n_pred) return HMLFC_E_CORRUPT;
                    T.n_flagged += (uint64_t)rr + (uint64_t)rp;
                    if (!T.pb.empty()) {
                        // block records (hmlfc_device.cuh): field widths and offsets of the plane's channels; .x counts the plane's bits
                        // until the prefix sum below turns it into the plane's first word
                        uint4 &pb = T.pb[k / 3];
                        const uint32_t w = m + (layout == 0 ? 0u : layout == 1 ? 2u : 3u);  // values < 2^m, 3 2^m, 5 2^m
                        pb.y |= w << (8 * c);
                        if (c == 0) pb.y |= D.mv_w << 24;
                        if (c < 2) pb.z |= ((uint32_t)offset & 0xFFFFu) << (16 * c); else pb.w = (uint32_t)offset & 0xFFFFu;
                        const uint64_t bits = (uint64_t)pb.x + (uint64_t)n_res * BB * w + (uint64_t)n_pred * D.mv_w;
                        if (bits > 0xFFFFFF00ull) return HMLFC_E_UNSUPPORTED;
                        pb.x = (uint32_t)bits;
                    }
                }
    if (!T.pb.empty()) {
        // slots: the six bit words of every group and the position of the group's first record in its plane
        for (uint64_t p = 0; p < n_pc / 3; ++p) {
            const uint4 pb = T.pb[p];
            const uint32_t w[3] = {pb.y & 0xFFu, (pb.y >> 8) & 0xFFu, (pb.y >> 16) & 0xFFu};
            uint64_t base = 0;
            for (int g = 0; g < D.fgroups; ++g) {
                const uint4 *fr = &T.flagrec[(p * (uint64_t)D.fgroups + (uint64_t)g) * 4];
                T.bslot[(p * (uint64_t)D.fgroups + (uint64_t)g) * 2] = make_uint4(fr[0].x, fr[1].x, fr[2].x, fr[0].z);
                T.bslot[(p * (uint64_t)D.fgroups + (uint64_t)g) * 2 + 1] = make_uint4(fr[1].z, fr[2].z, (uint32_t)base, 0u);
                for (int c = 0; c < 3; ++c)
                    base += (uint64_t)popcount32(fr[c].x) * BB * w[c] + (uint64_t)popcount32(fr[c].z) * D.mv_w;
            }
            if (base != (uint64_t)pb.x) return HMLFC_E_CORRUPT;  // (cannot happen: both count the same flags)
        }
        uint64_t word = 0;
        for (uint4 &pb : T.pb) {  // planes start at 32-byte boundaries
            const uint64_t words = ((uint64_t)pb.x + 31) / 32;
            if (word > 0xFFFFFF00ull) return HMLFC_E_UNSUPPORTED;
            pb.x = (uint32_t)word;
            word += (words + 7) & ~7ull;
        }
        T.brec_words = word + 8;  // fields are read as aligned 64-bit pairs plus one word
        if (T.brec_words > 0xFFFFFF00ull) return HMLFC_E_UNSUPPORTED;
    }

    // top-level RKVs: Y uint8 planes, then Co and Cg int16 LE planes -> short4 {Y, Co, Cg, 0} per full-resolution sample (subsampled
    // chroma is replicated here, once: nearest neighbour, R18)
    const uint8_t *py = s + off_rkv, *pco = py + n_top * npx, *pcg = pco + n_top * npx_c * 2;
    const uint64_t Wc = (uint64_t)(I.Ws >> D.cs);
    for (uint64_t q = 0; q < n_top; ++q)
        for (uint64_t y = 0; y < (uint64_t)I.Ht; ++y)
            for (uint64_t x = 0; x < (uint64_t)I.Ws; ++x) {
                const uint64_t i = q * npx + y * (uint64_t)I.Ws + x, ic = q * npx_c + (y >> D.cs) * Wc + (x >> D.cs);
                T.rkv[i] = make_short4((short)py[i], (short)(int16_t)rd16(pco + 2 * ic), (short)(int16_t)rd16(pcg + 2 * ic), 0);
            }
    return HMLFC_OK;
}

}  // namespace hmlfc
