// Fused decode + render kernel, CTA-per-tile variant with block-ROW tasks (sm_100a) -- the default of
// hmlfc_render for B = 4 streams.
//
// PAPER.md:289-293 (decoding procedure): "collect the required BISE compressed SRV blocks from the top level to
// the bottom level.  Using the block indices, we infer whether a block belongs to the predictive SRV images ...
// The motion vector values for the corresponding block are decoded"; "As a block of pixels are
// decoded, our method benefits any LF rendering scheme by providing fast access to neighboring pixels for
// interpolation"; PAPER.md:73 / :409 two-plane rendering.  Definitions: DESIGN.md sections 3 and 5.
//
// One CTA of 256 threads renders a 32 x 32 tile of one output view, 4 consecutive pixels per thread.  The cost of
// this path is instruction issue (profiles/), so the design minimises executed instructions per output pixel:
//   A   ray set-up (screen coordinates once per column / row, shared by shuffles), 16-tap footprint per pixel;
//   V   footprint box PER VIEW of the tile's (u,v) neighbourhood (warp reductions + a few shared atomics): a
//       tile that crosses a (u,v) cell boundary decodes each view only where its pixels need it;
//   T   warp 0 builds the tables: views -> cells, SRV planes of every level under the views ("slots"; a level-L
//       plane is shared by the 2^L x 2^L views below it and is decoded ONCE per tile), their boxes, offsets;
//   B1  one lane per (slot, channel, block row of the slot's box): the row's flag/rank words are loaded once
//       (128-bit records), non-empty blocks are compacted into a record list;
//   B2  one lane per record: the block's motion record (BISE decode_at, once per block) and the reference
//       plane's descriptor;
//   B3  one lane per (record, block row): the row's 4 stored values come from ONE pass over two 64-bit BISE
//       windows (plain / trit / quint without control flow); the motion-compensated reference row (two
//       neighbouring blocks of the reference SRV) likewise; written to the slot's int16 accumulator;
//   B4  one lane per (view, sample) cell: top-level RKV + the h per-level terms, inverse YCoCg-R, clamp ->
//       float RGB patch;
//   C   every pixel gathers its 16 taps from the patch (128-bit loads) and blends with packed fp32 FMAs.
// A tile whose tables do not fit the shared-memory arena (minification) is rendered as its four 16 x 16 quadrants,
// a quadrant that does not fit as four 8 x 8 sub-tiles, and an 8 x 8 sub-tile that still does not fit by 16 direct
// sample decodes per pixel.  All paths produce identical bytes.
#include "hmlfc_kernels.cuh"

namespace hmlfc {

namespace {

constexpr int kNT = 256;          // threads per CTA
constexpr int kTile = 32;         // tile edge in output pixels
constexpr int kPPL = 4;           // consecutive pixels per thread
constexpr int kMaxV = 4;          // views per axis of one tile's footprint
constexpr int kMaxViews = kMaxV * kMaxV;
constexpr int kMaxSlots = 52;     // 16 + 9 + 4 * 6 planes + slack
constexpr int kMaxChunks = 256;   // 32-cell chunks of the patch
constexpr int kSpecZero = 1536;   // 16-byte words of the accumulator region zeroed while warp 0 builds the tables
constexpr int kMinRec = 64;       // smallest record capacity worth starting with
constexpr uint32_t FULL = 0xffffffffu;
constexpr uint32_t kNone = 0xFFFFFFFFu;

// debug builds (-DHMLFC_PASS_STATS) count the passes of every size and why a pass was split
#ifdef HMLFC_PASS_STATS
__device__ unsigned long long g_pass_stats[64];  // [0..2] passes tried at 32/16/8, [3..5] passes done, [6] direct pixels passes, [8..] fail reasons, [16..] cycles of thread 0 per phase
__device__ long long g_phase_last[1 << 20];      // per CTA: clock of the previous mark
#define PASS_STAT(i) do { if (threadIdx.x == 0) atomicAdd(&g_pass_stats[i], 1ull); } while (0)
#define PHASE_MARK(i) do { if (threadIdx.x == 0) { const unsigned cta_ = (blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x; \
        const long long now_ = clock64(); if ((i) >= 0) atomicAdd(&g_pass_stats[16 + ((i) < 0 ? 0 : (i))], (unsigned long long)(now_ - g_phase_last[cta_ & ((1u << 20) - 1u)])); \
        g_phase_last[cta_ & ((1u << 20) - 1u)] = now_; } } while (0)
#else
#define PASS_STAT(i) do { } while (0)
#define PHASE_MARK(i) do { } while (0)
#endif


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

__device__ const DigitLut g_cta_digit_lut = make_digit_lut();

// n / d for n * d < 2^32 by one multiply-high (m == 0 encodes d <= 1)
__device__ __forceinline__ uint32_t magic_of(uint32_t d) { return d <= 1u ? 0u : 0xFFFFFFFFu / d + 1u; }
__device__ __forceinline__ uint32_t fdiv(uint32_t n, uint32_t m) { return m ? __umulhi(n, m) : n; }

struct ViewInfo {   // one view of the tile's (u,v) neighbourhood
    int s0, t0, ns, nt;          // footprint box of the view (ns == 0: no pixel of the tile touches it)
    int cellbase;                // first (view, sample) cell (a multiple of 32: a warp's cells belong to one view)
    uint32_t m_ns;               // magic multiplier of ns
    uint32_t rkv_lo, rkv_hi;     // index of the view's top-level RKV plane * Ht * Ws
};

struct SlotInfo {   // one SRV plane of one level under the tile's views
    uint32_t pc0, refpc0;        // descriptor index of channel 0 of the plane / of its cluster's reference plane
    int s0, t0, ns, s1;          // sample box (union of the boxes of the views below); s1 = last column
    int t1, bx0, by0, nbw;       // last row; block box
    int accbase, itembase, nbh;  // first accumulator sample; first B1 item (3 * nbh items); block rows
    uint32_t pred;               // plane is predictive
};

struct Ctl {
    int lo[4], hi[4];                    // (u0, v0) range of the tile's taps [0..1], unused [2..3]
    int vbox[kMaxViews][4];              // per view: min s, min t, max s, max t
    ViewInfo view[kMaxViews];
    SlotInfo slot[kMaxSlots + 1];
    int2 voff[kMaxViews][kMaxLevels];    // accumulator offset / row stride of the view's plane at level L
    int2 vcb[kMaxViews];                 // {cellbase - t0 * ns - s0, ns}: cell of sample (s,t) = x + t * y + s
    uint8_t chunkvw[kMaxChunks];         // view of the 32-cell chunk
    int lvl_base[kMaxLevels], lvl_pu0[kMaxLevels], lvl_pv0[kMaxLevels], lvl_nu[kMaxLevels];
    int nviews, nslots, ncell, nacc, nitems, reccap, fits;
    int n_rec, overflow;
    uint16_t lut[384];
};

struct PixTaps {  // one output pixel's 16-tap footprint
    uint32_t uv;  // u0 | v0 << 12 | du << 24 | dv << 25   (kNone: the ray misses the slab / pixel outside the view)
    uint32_t st;  // s0 | t0 << 14 | ds << 28 | dt << 29
    float fu, fv, fs, ft;
};

__device__ __forceinline__ uint32_t round_rgb(float r, float g, float b)
{
    const uint32_t R = (uint32_t)min(max(__float2int_rd(r + 0.5f), 0), 255);
    const uint32_t G = (uint32_t)min(max(__float2int_rd(g + 0.5f), 0), 255);
    const uint32_t B = (uint32_t)min(max(__float2int_rd(b + 0.5f), 0), 255);
    return R | (G << 8) | (B << 16);
}

// quadrilinear blend of 16 float RGB taps fetched by fetch(a, b): a = view (bit0 u, bit1 v), b = pixel (bit0 s, bit1 t)
template <typename Fetch>
__device__ __forceinline__ uint32_t blend16(const PixTaps &k, Fetch fetch)
{
    const float ws0 = 1.0f - k.fs, wt0 = 1.0f - k.ft, wu0 = 1.0f - k.fu, wv0 = 1.0f - k.fv;
    const float wst[4] = {ws0 * wt0, k.fs * wt0, ws0 * k.ft, k.fs * k.ft};
    const float wuv[4] = {wu0 * wv0, k.fu * wv0, wu0 * k.fv, k.fu * k.fv};
    float2 accRG = make_float2(0.f, 0.f), accB = make_float2(0.f, 0.f);
#pragma unroll
    for (int a = 0; a < 4; ++a) {
        float2 cRG = make_float2(0.f, 0.f), cB = make_float2(0.f, 0.f);
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const float4 t = fetch(a, b);
            const float2 w2 = make_float2(wst[b], wst[b]);
            cRG = __ffma2_rn(w2, make_float2(t.x, t.y), cRG);
            cB = __ffma2_rn(w2, make_float2(t.z, t.w), cB);
        }
        const float2 w2 = make_float2(wuv[a], wuv[a]);
        accRG = __ffma2_rn(w2, cRG, accRG);
        accB = __ffma2_rn(w2, cB, accB);
    }
    return round_rgb(accRG.x, accRG.y, accB.x);
}

// the tile does not fit even row by row (strong minification): 16 direct sample decodes
__device__ __noinline__ uint32_t direct_pixel(const DevStream &S, const PixTaps k)
{
    const int u0 = k.uv & 0xFFF, v0 = (k.uv >> 12) & 0xFFF, s0 = k.st & 0x3FFF, t0 = (k.st >> 14) & 0x3FFF;
    const int u1 = u0 + (int)((k.uv >> 24) & 1u), v1 = v0 + (int)((k.uv >> 25) & 1u);
    const int s1 = s0 + (int)((k.st >> 28) & 1u), t1 = t0 + (int)((k.st >> 29) & 1u);
    uint32_t c8[16];
#pragma unroll 1
    for (int a = 0; a < 16; ++a) c8[a] = decode_rgb8(S, (a & 4) ? u1 : u0, (a & 8) ? v1 : v0, (a & 1) ? s1 : s0, (a & 2) ? t1 : t0);
    return blend16(k, [&](int a, int b) {
        const uint32_t c = c8[a * 4 + b];
        return make_float4((float)(c & 0xFFu), (float)((c >> 8) & 0xFFu), (float)((c >> 16) & 0xFFu), 0.f);
    });
}

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

#ifndef HMLFC_ARENA_KB
#define HMLFC_ARENA_KB 68
#endif
#ifndef HMLFC_MINB
#define HMLFC_MINB 3
#endif
constexpr int kArenaDefault = HMLFC_ARENA_KB * 1024;  // 3 CTAs per SM: 3 x (68 KB + 6 KB static) of the 228 KB, up to 85 registers per thread.
// Measured (A/B on cfg2 / cfg3 / cfg4): 4 x 50 KB: 0.865 / 1.034 / 1.073 ms, 3 x 68 KB: 0.858 / 0.971 / 1.064 ms, 2 x 104 KB: 0.968 / 0.837 /
// 1.228 ms, 5 x 38 KB: 1.062 / 1.218 / 1.321 ms -- the kernel is not occupancy-bound; fewer spills and fewer split tiles win.
constexpr int kMinBlocksDefault = HMLFC_MINB;
// Second instance for views that look at about as many light-field samples as they have pixels (cfg3: 512^2 views of 512^2 images):
// 2 CTAs per SM with 104 KB each, so that far fewer tiles have to be split into 16 x 16 / 8 x 8 passes (cfg3: 0.97 -> 0.84 ms).  The
// launcher picks it from the sizes alone: output pixels per view < 2 x light-field pixels per view (a hint: both give the same bytes).
#ifndef HMLFC_ARENA_BIG_KB
#define HMLFC_ARENA_BIG_KB 104
#endif
constexpr int kArenaBig = HMLFC_ARENA_BIG_KB * 1024;
constexpr int kMinBlocksBig = 2;
// Third instance for strong magnification (cfg5: 2048^2 views of 640^2 images, a tile looks at few samples): 4 CTAs x 50 KB, <= 64 registers.
constexpr int kArenaSmall = 50 * 1024;
constexpr int kMinBlocksSmall = 4;
#ifndef HMLFC_EST_SLACK
#define HMLFC_EST_SLACK 120
#endif
constexpr int kEstSlackPct = HMLFC_EST_SLACK;  // the 32 x 32 pass is tried when the estimate is below this share of the arena

// ---------------------------------------------------------------------------------------------------------------
// Phases T, B1-B4 for the sub-tile whose (u,v) range (ctl.lo / ctl.hi) and per-view footprint boxes (ctl.vbox) are
// set: builds the tables and, if they fit the arena, the float RGB patch of every (view, sample) cell.  Returns
// false (CTA-uniform) when the sub-tile does not fit; the caller then splits it.  Called by all 256 threads.
#ifndef HMLFC_BP_ATTR
#define HMLFC_BP_ATTR __forceinline__
#endif
template <int kArenaBytes>
__device__ HMLFC_BP_ATTR bool build_patch(const DevStream &S, Ctl &ctl, unsigned char *__restrict__ arena)
{
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int h = S.h;
    const int bu0 = ctl.lo[0], bv0 = ctl.lo[1];
    const int nu = ctl.hi[0] - bu0 + 1, nv = ctl.hi[1] - bv0 + 1;

    // -------------------------------------------------------- T: tables (warp 0)
    if (warp == 0) {
        const int nviews = nu * nv;
        int vs0 = 0, vt0 = 0, vns = 0, vnt = 0;
        if (lane < nviews && ctl.vbox[lane][2] >= 0) {
            vs0 = ctl.vbox[lane][0]; vt0 = ctl.vbox[lane][1];
            vns = ctl.vbox[lane][2] - vs0 + 1; vnt = ctl.vbox[lane][3] - vt0 + 1;
        }
        const int vcells = (vns * vnt + 31) & ~31;  // whole warps per view
        int incl = vcells;
#pragma unroll
        for (int o = 1; o < kMaxViews; o <<= 1) {
            const int n = __shfl_up_sync(FULL, incl, o);
            if (lane >= o) incl += n;
        }
        const int ncell = __shfl_sync(FULL, incl, kMaxViews - 1);
        if (lane < kMaxViews) {
            ViewInfo vi;
            vi.s0 = vs0; vi.t0 = vt0; vi.ns = vns; vi.nt = vnt;
            vi.cellbase = incl - vcells;
            ctl.vcb[lane] = make_int2(vi.cellbase - vt0 * vns - vs0, vns);
            for (int c = vi.cellbase >> 5; c < min(incl >> 5, kMaxChunks); ++c) ctl.chunkvw[c] = (uint8_t)lane;
            vi.m_ns = magic_of((uint32_t)vns);
            const int iv = lane / nu, iu = lane - iv * nu;
            const unsigned long long ro = (unsigned long long)(((bv0 + iv) >> h) * S.UH + ((bu0 + iu) >> h)) *
                                          (unsigned long long)S.Ht * (unsigned long long)S.Ws;
            vi.rkv_lo = (uint32_t)ro; vi.rkv_hi = (uint32_t)(ro >> 32);
            ctl.view[lane] = vi;
        }
        // per level the rectangle of planes over the views; lane L owns level L
        int pu0 = 0, pv0 = 0, nuL = 0, cntL = 0;
        if (lane >= S.lmin && lane < h) {  // progressive decoding: no planes below lmin
            pu0 = bu0 >> lane; pv0 = bv0 >> lane;
            nuL = ((bu0 + nu - 1) >> lane) - pu0 + 1;
            cntL = nuL * (((bv0 + nv - 1) >> lane) - pv0 + 1);
        }
        int lincl = cntL;
#pragma unroll
        for (int o = 1; o < kMaxLevels; o <<= 1) {
            const int n = __shfl_up_sync(FULL, lincl, o);
            if (lane >= o) lincl += n;
        }
        const int nslots = __shfl_sync(FULL, lincl, h - 1);
        if (lane < h) { ctl.lvl_base[lane] = lincl - cntL; ctl.lvl_pu0[lane] = pu0; ctl.lvl_pv0[lane] = pv0; ctl.lvl_nu[lane] = nuL; }
        __syncwarp();
        int accrun = 0, itemrun = 0;
        if (nslots <= kMaxSlots) {
            for (int sb = 0; sb < nslots; sb += 32) {
                const int s = sb + lane;
                SlotInfo si;
                si.pc0 = si.refpc0 = 0u; si.pred = 0u;
                si.s0 = si.t0 = 0; si.ns = 0; si.s1 = si.t1 = -1; si.bx0 = si.by0 = 0; si.nbw = 0; si.nbh = 0;
                int nsamp = 0;
                if (s < nslots) {
                    int L = 0;
                    while (L + 1 < h && s >= ctl.lvl_base[L + 1]) ++L;
                    const int jj = s - ctl.lvl_base[L], n = ctl.lvl_nu[L];
                    const int jv = jj / n;
                    const int pv = ctl.lvl_pv0[L] + jv, pu = ctl.lvl_pu0[L] + (jj - jv * n);
                    const LevelDesc lv = S.lev[L];
                    si.pc0 = lv.pc_base + (uint32_t)(pv * lv.UL + pu) * 3u;
                    si.refpc0 = lv.pc_base + (uint32_t)((pv & ~1) * lv.UL + (pu & ~1)) * 3u;
                    si.pred = (uint32_t)((pu | pv) & 1);
                    // union of the boxes of the views below this plane
                    const int iu0 = max(pu << L, bu0) - bu0, iu1 = min(((pu + 1) << L) - 1, bu0 + nu - 1) - bu0;
                    const int iv0 = max(pv << L, bv0) - bv0, iv1 = min(((pv + 1) << L) - 1, bv0 + nv - 1) - bv0;
                    int a0 = 0x7fffffff, a1 = 0x7fffffff, a2 = -1, a3 = -1;
                    for (int iv = iv0; iv <= iv1; ++iv)
                        for (int iu = iu0; iu <= iu1; ++iu) {
                            const int vw = iv * nu + iu;
                            if (ctl.vbox[vw][2] >= 0) {
                                a0 = min(a0, ctl.vbox[vw][0]); a1 = min(a1, ctl.vbox[vw][1]);
                                a2 = max(a2, ctl.vbox[vw][2]); a3 = max(a3, ctl.vbox[vw][3]);
                            }
                        }
                    if (a2 >= 0) {
                        si.s0 = a0; si.t0 = a1; si.s1 = a2; si.t1 = a3; si.ns = a2 - a0 + 1;
                        si.bx0 = a0 >> 2; si.by0 = a1 >> 2;
                        si.nbw = (a2 >> 2) - si.bx0 + 1; si.nbh = (a3 >> 2) - si.by0 + 1;
                        nsamp = si.ns * (a3 - a1 + 1);
                    }
                }
                int ai = nsamp, ii = 3 * si.nbh;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int n1 = __shfl_up_sync(FULL, ai, o), n2 = __shfl_up_sync(FULL, ii, o);
                    if (lane >= o) { ai += n1; ii += n2; }
                }
                si.accbase = accrun + ai - nsamp;
                si.itembase = itemrun + ii - 3 * si.nbh;
                if (s < nslots) ctl.slot[s] = si;
                accrun += __shfl_sync(FULL, ai, 31);
                itemrun += __shfl_sync(FULL, ii, 31);
            }
        }
        if (lane == 0) {
            // accumulators (8 bytes per slot sample), then the patch (16 bytes per cell) aliased by the record list (32 bytes each)
            const long long accbytes = ((long long)accrun * 8 + 15) & ~15LL;
            const long long rest = (long long)kArenaBytes - accbytes;
            const bool fits = nslots <= kMaxSlots && ncell <= 32 * kMaxChunks && rest >= (long long)ncell * 16 && rest >= (long long)kMinRec * 32;
            ctl.nviews = nviews; ctl.nslots = nslots; ctl.ncell = ncell; ctl.nacc = accrun; ctl.nitems = itemrun;
            ctl.reccap = fits ? (int)min(rest / 32, 65535LL) : 0;
            ctl.fits = fits ? 1 : 0;
            if (nslots <= kMaxSlots) ctl.slot[nslots].itembase = itemrun;  // sentinel of the item -> slot search
        }
    } else {
        // meanwhile the other warps zero the head of the accumulator region (its size is not known yet)
        uint4 *z = reinterpret_cast<uint4 *>(arena);
        for (int q = tid - 32; q < kSpecZero; q += kNT - 32) z[q] = make_uint4(0u, 0u, 0u, 0u);
    }
    __syncthreads();
    PHASE_MARK(4);
    if (!ctl.fits) { PASS_STAT(10); return false; }

    const int nviews = ctl.nviews, ncell = ctl.ncell, nacc = ctl.nacc, nitems = ctl.nitems, reccap = ctl.reccap;
    uint2 *acc = reinterpret_cast<uint2 *>(arena);
    unsigned char *region2 = arena + (((size_t)nacc * 8 + 15) & ~(size_t)15);
    uint4 *rec = reinterpret_cast<uint4 *>(region2);      // [reccap][2]
    float4 *patch = reinterpret_cast<float4 *>(region2);  // [ncell], after the records are dead
    // ---------------------------------------------------- zero the accumulators; accumulator offsets of every (view, level)
    {
        uint4 *z = reinterpret_cast<uint4 *>(arena);
        const int nz = (nacc + 1) >> 1;
        for (int q = kSpecZero + tid; q < nz; q += kNT) z[q] = make_uint4(0u, 0u, 0u, 0u);  // the rest (warps 1..7 zeroed the head during T)
        for (int q = tid; q < nviews * h; q += kNT) {
            const int vw = q / h, L = q - vw * h;
            if (L < S.lmin) continue;
            const int iv = vw / nu, iu = vw - iv * nu;
            const int sidx = ctl.lvl_base[L] + (((bv0 + iv) >> L) - ctl.lvl_pv0[L]) * ctl.lvl_nu[L] + (((bu0 + iu) >> L) - ctl.lvl_pu0[L]);
            const SlotInfo &sl = ctl.slot[sidx];
            const ViewInfo &vi = ctl.view[vw];
            ctl.voff[vw][L] = make_int2(sl.accbase + (vi.t0 - sl.t0) * sl.ns + (vi.s0 - sl.s0), sl.ns);
        }
    }
    // ---------------------------------------------------- B1: one lane per (slot, channel, block row): flag words -> records
    for (int base = 0; base < nitems; base += kNT) {
        const int it = base + tid;
        const bool on = it < nitems;
        uint4 d = make_uint4(0u, 0u, 0u, 0u);
        uint32_t refpc = 0u, sc = 0u, pred = 0u;
        int b0 = 0, b1 = -1, by = 0, rowb = 0;
        size_t frbase = 0;
        if (on) {
            int s = 0;
            while (it >= ctl.slot[s + 1].itembase) ++s;
            const SlotInfo &sl = ctl.slot[s];
            const int r = it - sl.itembase;
            const int c = r / sl.nbh, jr = r - c * sl.nbh;
            d = ldg(S.pc + sl.pc0 + c);
            frbase = flag_index(S, sl.pc0 + (uint32_t)c, 0u);  // = d.x, without waiting for d
            refpc = sl.refpc0 + (uint32_t)c;
            sc = ((uint32_t)s << 22) | ((uint32_t)c << 28);
            pred = sl.pred;
            by = sl.by0 + jr;
            rowb = by * S.nbx;
            b0 = rowb + sl.bx0; b1 = b0 + sl.nbw - 1;
        }
        const int ng = on ? (b1 >> 5) - (b0 >> 5) + 1 : 0;
        const int ngmax = __reduce_max_sync(FULL, ng);
        for (int gi = 0; gi < ngmax; ++gi) {
            uint32_t resb = 0u, prdb = 0u;
            uint4 fr = make_uint4(0u, 0u, 0u, 0u);
            const int g = (b0 >> 5) + gi;
            if (gi < ng) {
                fr = ldg(S.flagrec + frbase + 4u * (size_t)g);
                const int lo = max(b0 - (g << 5), 0), hi = min(b1 - (g << 5), 31);
                const uint32_t mask = (0xFFFFFFFFu >> (31 - hi)) & (0xFFFFFFFFu << lo);
                resb = fr.x & mask;
                prdb = pred ? (fr.z & mask) : 0u;
            }
            uint32_t any = resb | prdb;
            const int cnt = (int)popc(any);
            int inc = cnt;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int n = __shfl_up_sync(FULL, inc, o);
                if (lane >= o) inc += n;
            }
            const int tot = __shfl_sync(FULL, inc, 31);
            if (tot == 0) continue;
            int wbase = 0;
            if (lane == 31) wbase = atomicAdd(&ctl.n_rec, tot);
            wbase = __shfl_sync(FULL, wbase, 31);
            int idx = wbase + inc - cnt;
            while (any) {
                const int bp = __ffs(any) - 1;
                const uint32_t bit = 1u << bp;
                any &= any - 1u;
                const bool hr = (resb & bit) != 0u, hp = (prdb & bit) != 0u;
                if (idx < reccap) {
                    // own payload base, rank * 16, descriptor word, rank of the motion record | MV string base, reference pc, slot / channel, block position
                    rec[2 * idx] = make_uint4(d.y, hr ? ((fr.y + popc(fr.x & (bit - 1u))) << 4) : kNone, d.w,
                                              hp ? (fr.w + popc(fr.z & (bit - 1u))) : kNone);
                    rec[2 * idx + 1] = make_uint4(d.z, refpc, sc, (uint32_t)((g << 5) + bp - rowb) | ((uint32_t)by << 16));
                } else {
                    ctl.overflow = 1;
                }
                ++idx;
            }
        }
    }
    __syncthreads();
    PHASE_MARK(5);
    if (ctl.overflow != 0) { PASS_STAT(11); return false; }
    const int nrec = ctl.n_rec;
    // ------------------------------------------------ B2: motion record + reference descriptor, once per block
    for (int rr = tid; rr < nrec; rr += kNT) {
        const uint4 r0 = rec[2 * rr], r1 = rec[2 * rr + 1];
        if (r0.w != kNone) {
            const uint32_t mr = bise_at(S.mv + r1.x, r0.w, S.mv_layout, S.mv_m, ctl.lut);
            int md, dx, dy;
            mv_unpack(S, mr, md, dx, dy);
            const uint4 dr = ldg(S.pc + r1.y);
            rec[2 * rr].w = 0x80000000u | ((uint32_t)md << 16) | ((uint32_t)(dx + S.W) << 8) | (uint32_t)(dy + S.W);
            rec[2 * rr + 1] = make_uint4(dr.x, dr.y, r1.z | (dr.w & 0x3FFFFFu), r1.w);
        } else {
            rec[2 * rr].w = 0u;
            rec[2 * rr + 1] = make_uint4(0u, 0u, r1.z, r1.w);
        }
    }
    __syncthreads();
    PHASE_MARK(6);
    // ------------------------------------------------ B3: one lane per (record, block row): 4 stored / re-compensated values
    int16_t *acc16 = reinterpret_cast<int16_t *>(arena);
    for (int t = tid; t < 4 * nrec; t += kNT) {
        const int rr = t >> 2, ky = t & 3;
        const uint4 r0 = rec[2 * rr], r1 = rec[2 * rr + 1];
        const SlotInfo &sl = ctl.slot[(r1.z >> 22) & 63u];
        const int yy = (int)((r1.w >> 16) << 2) + ky;
        const int st0 = sl.t0, st1 = sl.t1;
        if (yy < st0 || yy > st1) continue;
        const int xx = (int)((r1.w & 0xFFFFu) << 2);
        uint2 own = make_uint2(0u, 0u);
        if (r0.y != kNone) own = bise_row4(S.pay + r0.x, r0.y + (uint32_t)(ky << 2), r0.z, ctl.lut);
        int e0 = (int)(int16_t)(own.x & 0xFFFFu), e1 = (int)own.x >> 16, e2 = (int)(int16_t)(own.y & 0xFFFFu), e3 = (int)own.y >> 16;
        if (r0.w) {
            const int rx = xx + (int)((r0.w >> 8) & 0xFFu) - S.W, ry = yy + (int)(r0.w & 0xFFu) - S.W;
            if ((unsigned)ry < (unsigned)S.Ht) {
                // the 4 reference samples (rx .. rx+3, ry) lie in the block row ry>>2, blocks rx>>2 and (rx>>2)+1
                const int o = rx & 3, bxa = rx >> 2;
                const uint32_t i0 = (uint32_t)((ry & 3) << 2);
                const int rowb = (ry >> 2) * S.nbx;
                uint2 qa = make_uint2(0u, 0u), qb = make_uint2(0u, 0u);
                if ((unsigned)bxa < (unsigned)S.nbx) {
                    const int b = rowb + bxa;
                    const uint4 fr = ldg(S.flagrec + r1.x + 4u * (uint32_t)(b >> 5));
                    const uint32_t bit = 1u << (b & 31);
                    if (fr.x & bit) qa = bise_row4(S.pay + r1.y, ((fr.y + popc(fr.x & (bit - 1u))) << 4) + i0, r1.z, ctl.lut);
                }
                if (o && (unsigned)(bxa + 1) < (unsigned)S.nbx) {
                    const int b = rowb + bxa + 1;
                    const uint4 fr = ldg(S.flagrec + r1.x + 4u * (uint32_t)(b >> 5));
                    const uint32_t bit = 1u << (b & 31);
                    if (fr.x & bit) qb = bise_row4(S.pay + r1.y, ((fr.y + popc(fr.x & (bit - 1u))) << 4) + i0, r1.z, ctl.lut);
                }
                // samples o .. o+3 of the 8-sample string qa | qb
                uint32_t w0 = qa.x, w1 = qa.y, w2 = qb.x, w3 = qb.y;
                if (o & 2) { w0 = w1; w1 = w2; w2 = w3; }
                const uint32_t sh = (uint32_t)(o & 1) << 4;
                const uint32_t q01 = __funnelshift_r(w0, w1, sh), q23 = __funnelshift_r(w1, w2, sh);
                const int q0 = (int)(int16_t)(q01 & 0xFFFFu), q1 = (int)q01 >> 16, q2 = (int)(int16_t)(q23 & 0xFFFFu), q3 = (int)q23 >> 16;
                // R10: subtractive P = e + R, additive P = e - R
                if (r0.w & 0x10000u) { e0 -= q0; e1 -= q1; e2 -= q2; e3 -= q3; }
                else { e0 += q0; e1 += q1; e2 += q2; e3 += q3; }
            }
        }
        const int c = (int)((r1.z >> 28) & 3u);
        int16_t *dst = acc16 + (((sl.accbase + (yy - st0) * sl.ns + (xx - sl.s0)) << 2) + c);
        const int ss0 = sl.s0, ss1 = sl.s1;
        if (xx >= ss0 && xx <= ss1) dst[0] = (int16_t)e0;
        if (xx + 1 >= ss0 && xx + 1 <= ss1) dst[4] = (int16_t)e1;
        if (xx + 2 >= ss0 && xx + 2 <= ss1) dst[8] = (int16_t)e2;
        if (xx + 3 >= ss0 && xx + 3 <= ss1) dst[12] = (int16_t)e3;
    }
    __syncthreads();
    PHASE_MARK(7);
    // ------------------------------------------------ B4: top-level RKV + per-level terms -> float RGB patch
    for (int q = tid; q < ncell; q += kNT) {
        const int vw = ctl.chunkvw[q >> 5];
        const ViewInfo vi = ctl.view[vw];
        const uint32_t local = (uint32_t)(q - vi.cellbase);
        const uint32_t it = fdiv(local, vi.m_ns), is = local - it * (uint32_t)vi.ns;
        if ((int)it >= vi.nt) continue;  // padding of the view's last chunk
        const unsigned long long ro = ((unsigned long long)vi.rkv_hi << 32) | vi.rkv_lo;
        const short4 rk = ldg(S.rkv + ro + (uint32_t)((vi.t0 + (int)it) * S.Ws + vi.s0 + (int)is));
        int a[3] = {rk.x, rk.y, rk.z};
        for (int L = S.lmin; L < h; ++L) {
            const int2 vo = ctl.voff[vw][L];
            const uint2 w = acc[vo.x + (int)it * vo.y + (int)is];
            a[0] += (int)(int16_t)(w.x & 0xFFFFu);
            a[1] += (int)w.x >> 16;
            a[2] += (int)(int16_t)(w.y & 0xFFFFu);
        }
        const uint32_t c8 = ycocg_to_rgb8(a);
        // the patch aliases the record list: all B3 readers passed the barrier above
        patch[q] = make_float4((float)(c8 & 0xFFu), (float)((c8 >> 8) & 0xFFu), (float)((c8 >> 16) & 0xFFu), 0.f);
    }
    __syncthreads();
    PHASE_MARK(8);
    return true;
}

// ---------------------------------------------------------------------------------------------------------------
// Pixel mapping of a pass.  ts = 32: the whole tile, thread (tid & 7, tid >> 3) owns 4 consecutive pixels.  ts = 16 /
// 8: a sub-tile, one pixel per thread (pixel slot 0; ts = 8 uses the first 64 threads).  One code path serves both
// (slots 1..3 are simply empty in sub-tile passes): the kernel is instruction-cache sensitive, so the phases exist once.
__device__ __forceinline__ void thread_pixel(int ox, int oy, int ts, int &x0, int &y, int &npix)
{
    const int tid = threadIdx.x;
    if (ts == kTile) { x0 = ox + (tid & 7) * kPPL; y = oy + (tid >> 3); npix = kPPL; }
    else { const int sh = ts == 16 ? 4 : 3; x0 = ox + (tid & (ts - 1)); y = oy + (tid >> sh); npix = tid < ts * ts ? 1 : 0; }
}

// ---------------------------------------------------------------- A: rays of the thread's pixels
__device__ __forceinline__ void setup_rays(const DevStream &S, const Camera &cam, int W, int H, int ox, int oy, int ts, PixTaps (&pt)[kPPL])
{
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    int x0, y, npix;
    thread_pixel(ox, oy, ts, x0, y, npix);
    // screen coordinates once per column / row of the tile, shared by shuffles (sub-tiles: each lane its own)
    const float pxl = ray_screen(cam.tan_half_x, W, ts == kTile ? ox + lane : x0);
    const float pyl = ray_screen(cam.tan_half_y, H, ts == kTile ? oy + warp * 4 + (lane & 3) : y);
    const float py = __shfl_sync(FULL, pyl, ts == kTile ? lane >> 3 : lane);
#pragma unroll
    for (int p = 0; p < kPPL; ++p) {
        const float px = __shfl_sync(FULL, pxl, ts == kTile ? (tid & 7) * kPPL + p : lane);
        pt[p].uv = kNone; pt[p].st = 0u;
        pt[p].fu = pt[p].fv = pt[p].fs = pt[p].ft = 0.f;
        if (p < npix && x0 + p < W && y < H) {
            const Ray r = ray_from_screen(S, cam, px, py);
            if (r.hit) {
                const Taps k = tap_setup(S, r);
                pt[p].uv = (uint32_t)k.u0 | ((uint32_t)k.v0 << 12) | ((uint32_t)(k.u1 - k.u0) << 24) | ((uint32_t)(k.v1 - k.v0) << 25);
                pt[p].st = (uint32_t)k.s0 | ((uint32_t)k.t0 << 14) | ((uint32_t)(k.s1 - k.s0) << 28) | ((uint32_t)(k.t1 - k.t0) << 29);
                pt[p].fu = k.fu; pt[p].fv = k.fv; pt[p].fs = k.fs; pt[p].ft = k.ft;
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// One pass over a (sub-)tile whose rays are set up: footprint boxes (V), tables + decode (build_patch), gather + blend
// (C).  Returns true (CTA-uniform) when rgb[] holds the pass's pixels (background where the ray misses); false
// when the tables do not fit the arena and the (sub-)tile must be split.
template <int kArenaBytes>
__device__ __forceinline__ bool tile_pass(const DevStream &S, Ctl &ctl, unsigned char *__restrict__ arena, const PixTaps (&pt)[kPPL],
                                          uint32_t (&rgb)[kPPL])
{
    constexpr int PPL = kPPL;
    const int tid = threadIdx.x, lane = tid & 31;
    __syncthreads();  // the previous pass's readers of ctl / the patch are done (and the digit table is loaded)
    if (tid < kMaxViews) { ctl.vbox[tid][0] = 0x7fffffff; ctl.vbox[tid][1] = 0x7fffffff; ctl.vbox[tid][2] = -1; ctl.vbox[tid][3] = -1; }
    if (tid < 4) { ctl.lo[tid] = 0x7fffffff; ctl.hi[tid] = -1; }
    if (tid == 0) { ctl.n_rec = 0; ctl.overflow = 0; ctl.fits = 0; }
    __syncthreads();
    PHASE_MARK(1);

    // ------------------------------------------------------------ lane summary: common (u0, v0, du, dv) key and (s,t) box of the lane's pixels
    uint32_t key = kNone;
    bool mixed = false;
    int ls0 = 0x7fffffff, lt0 = 0x7fffffff, ls1 = -1, lt1 = -1;
    int ulo = 0x7fffffff, vlo = 0x7fffffff, uhi = -1, vhi = -1;
#pragma unroll
    for (int p = 0; p < PPL; ++p)
        if (pt[p].uv != kNone) {
            if (key == kNone) key = pt[p].uv;
            else if (pt[p].uv != key) mixed = true;
            const int s0 = pt[p].st & 0x3FFF, t0 = (pt[p].st >> 14) & 0x3FFF;
            ls0 = min(ls0, s0); ls1 = max(ls1, s0 + (int)((pt[p].st >> 28) & 1u));
            lt0 = min(lt0, t0); lt1 = max(lt1, t0 + (int)((pt[p].st >> 29) & 1u));
            const int u0 = pt[p].uv & 0xFFF, v0 = (pt[p].uv >> 12) & 0xFFF;
            ulo = min(ulo, u0); uhi = max(uhi, u0 + (int)((pt[p].uv >> 24) & 1u));
            vlo = min(vlo, v0); vhi = max(vhi, v0 + (int)((pt[p].uv >> 25) & 1u));
        }
    ulo = __reduce_min_sync(FULL, ulo); vlo = __reduce_min_sync(FULL, vlo);
    uhi = __reduce_max_sync(FULL, uhi); vhi = __reduce_max_sync(FULL, vhi);
    const int ws0 = __reduce_min_sync(FULL, ls0), wt0 = __reduce_min_sync(FULL, lt0);
    const int ws1 = __reduce_max_sync(FULL, ls1), wt1 = __reduce_max_sync(FULL, lt1);
    if (lane == 0 && uhi >= 0) {
        atomicMin(&ctl.lo[0], ulo); atomicMin(&ctl.lo[1], vlo); atomicMin(&ctl.lo[2], ws0); atomicMin(&ctl.lo[3], wt0);
        atomicMax(&ctl.hi[0], uhi); atomicMax(&ctl.hi[1], vhi); atomicMax(&ctl.hi[2], ws1); atomicMax(&ctl.hi[3], wt1);
    }
    __syncthreads();
    PHASE_MARK(2);
    const int bu0 = ctl.lo[0], bv0 = ctl.lo[1];
    const int nu = ctl.hi[0] - bu0 + 1, nv = ctl.hi[1] - bv0 + 1;
    if (ctl.hi[0] < 0) return true;  // no ray of the sub-tile hits the slab: background only
    if (nu > kMaxV || nv > kMaxV) { PASS_STAT(8); return false; }
    {
        // Early exit before the tables are built: from the pass's exact (u,v) range and (s,t) box, cells ~ (2 ns + nu)
        // (2 nt + nv) (every pixel touches 2 x 2 views) and accumulator samples ~ cells (level 0) + box area x planes
        // of every level >= 1.  Only a hint (build_patch decides): a pass that is let through and does not fit is
        // split after the tables are built, one that is split needlessly costs some halo.
        const int ns = ctl.hi[2] - ctl.lo[2] + 1, nt = ctl.hi[3] - ctl.lo[3] + 1;
        const int area = ns * nt;
        const int cells = (2 * ns + nu) * (2 * nt + nv) + 16 * nu * nv;
        int accs = cells;
        for (int L = 1; L < S.h; ++L)
            accs += area * ((((bu0 + nu - 1) >> L) - (bu0 >> L) + 1) * (((bv0 + nv - 1) >> L) - (bv0 >> L) + 1));
        if (16 * cells + 8 * accs > kArenaBytes * kEstSlackPct / 100) { PASS_STAT(9); return false; }
    }

    // -------------------------------------------------------- V: footprint box per view
    // lanes with one common key first (the usual case: one or two rounds per warp), then pixel by pixel
    auto merge_boxes = [&](uint32_t k, int a0, int a1, int a2, int a3) {
        uint32_t todo = __ballot_sync(FULL, k != kNone);
        while (todo) {
            const int leader = __ffs(todo) - 1;
            const uint32_t kk = __shfl_sync(FULL, k, leader);
            const bool mine = k == kk;
            const int m0 = __reduce_min_sync(FULL, mine ? a0 : 0x7fffffff), m1 = __reduce_min_sync(FULL, mine ? a1 : 0x7fffffff);
            const int m2 = __reduce_max_sync(FULL, mine ? a2 : -1), m3 = __reduce_max_sync(FULL, mine ? a3 : -1);
            if (lane < 4) {
                const int du = (int)((kk >> 24) & 1u), dv = (int)((kk >> 25) & 1u);
                const int au = lane & 1, av = lane >> 1;
                if ((!au || du) && (!av || dv)) {
                    const int vw = ((int)((kk >> 12) & 0xFFF) - bv0 + av) * nu + ((int)(kk & 0xFFF) - bu0 + au);
                    atomicMin(&ctl.vbox[vw][0], m0); atomicMin(&ctl.vbox[vw][1], m1);
                    atomicMax(&ctl.vbox[vw][2], m2); atomicMax(&ctl.vbox[vw][3], m3);
                }
            }
            todo &= ~__ballot_sync(FULL, mine);
        }
    };
    merge_boxes(mixed ? kNone : key, ls0, lt0, ls1, lt1);
    if (PPL > 1 && __any_sync(FULL, mixed)) {
#pragma unroll
        for (int p = 0; p < PPL; ++p) {
            const int s0 = pt[p].st & 0x3FFF, t0 = (pt[p].st >> 14) & 0x3FFF;
            merge_boxes(mixed ? pt[p].uv : kNone, s0, t0, s0 + (int)((pt[p].st >> 28) & 1u), t0 + (int)((pt[p].st >> 29) & 1u));
        }
    }
    __syncthreads();
    PHASE_MARK(3);

    if (!build_patch<kArenaBytes>(S, ctl, arena)) return false;

    // ------------------------------------------------ C: gather + blend
    const float4 *patch = reinterpret_cast<const float4 *>(arena + (((size_t)ctl.nacc * 8 + 15) & ~(size_t)15));
#pragma unroll
    for (int p = 0; p < PPL; ++p)
        if (pt[p].uv != kNone) {
            const int iu = (int)(pt[p].uv & 0xFFF) - bu0, iv = (int)((pt[p].uv >> 12) & 0xFFF) - bv0;
            const int s0 = (int)(pt[p].st & 0x3FFF), t0 = (int)((pt[p].st >> 14) & 0x3FFF);
            const int du = (int)((pt[p].uv >> 24) & 1u), dv = ((pt[p].uv >> 25) & 1u) ? nu : 0;
            const int ds = (int)((pt[p].st >> 28) & 1u), dt = (int)((pt[p].st >> 29) & 1u);
            const int vw0 = iv * nu + iu;
            int vb[4], vs[4];
#pragma unroll
            for (int a = 0; a < 4; ++a) {
                const int2 cb = ctl.vcb[vw0 + ((a & 1) ? du : 0) + ((a & 2) ? dv : 0)];
                vb[a] = cb.x + t0 * cb.y + s0;
                vs[a] = dt ? cb.y : 0;
            }
            rgb[p] = blend16(pt[p], [&](int a, int b) { return patch[vb[a] + ((b & 1) ? ds : 0) + ((b & 2) ? vs[a] : 0)]; });
        }
    PHASE_MARK(9);
    return true;
}

// ---------------------------------------------------------------- stores
__device__ __forceinline__ void store4(uint8_t *__restrict__ out, int view, int W, int H, int x0, int y, const uint32_t (&rgb)[4], int out_aligned)
{
    if (y >= H || x0 >= W) return;
    uint8_t *o = out + 3 * (((size_t)view * H + (size_t)y) * (size_t)W + (size_t)x0);
    if (out_aligned && x0 + 4 <= W) {  // 12 contiguous bytes per thread
        uint32_t *o32 = reinterpret_cast<uint32_t *>(o);
        o32[0] = rgb[0] | (rgb[1] << 24);
        o32[1] = (rgb[1] >> 8) | (rgb[2] << 16);
        o32[2] = (rgb[2] >> 16) | (rgb[3] << 8);
    } else {
#pragma unroll
        for (int p = 0; p < 4; ++p)
            if (x0 + p < W) {
                o[3 * p + 0] = (uint8_t)(rgb[p] & 0xFF);
                o[3 * p + 1] = (uint8_t)((rgb[p] >> 8) & 0xFF);
                o[3 * p + 2] = (uint8_t)((rgb[p] >> 16) & 0xFF);
            }
    }
}

// one pixel per lane, 4 consecutive lanes = 4 consecutive pixels of a row: their 12 bytes leave as three 32-bit words
__device__ __forceinline__ void store1(uint8_t *__restrict__ out, int view, int W, int H, int x, int y, bool active, uint32_t rgb, int out_aligned)
{
    const uint32_t nb = __shfl_down_sync(FULL, rgb, 1);
    if (!active || y >= H || x >= W) return;
    uint8_t *o = out + 3 * (((size_t)view * H + (size_t)y) * (size_t)W + (size_t)x);
    if (out_aligned) {  // W % 4 == 0 and x % 4 == lane % 4: the group's 4 pixels are all inside the view
        const int j = x & 3;
        if (j < 3) {
            const uint32_t w = j == 0 ? (rgb | (nb << 24)) : j == 1 ? ((rgb >> 8) | (nb << 16)) : ((rgb >> 16) | (nb << 8));
            reinterpret_cast<uint32_t *>(o - 3 * j)[j] = w;
        }
    } else {
        o[0] = (uint8_t)(rgb & 0xFF);
        o[1] = (uint8_t)((rgb >> 8) & 0xFF);
        o[2] = (uint8_t)((rgb >> 16) & 0xFF);
    }
}

template <int kArenaBytes, int kMinBlocks>
__global__ void __launch_bounds__(kNT, kMinBlocks)
render_cta_kernel(const __grid_constant__ DevStream S, const Camera *__restrict__ cams, int W, int H, uint8_t *__restrict__ out, int out_aligned)
{
    extern __shared__ __align__(16) unsigned char arena[];
    __shared__ Ctl ctl;
    const int tid = threadIdx.x;
    const int ox = blockIdx.x * kTile, oy = blockIdx.y * kTile;
    const int view = blockIdx.z;

    for (int q = tid; q < 192; q += kNT)
        reinterpret_cast<uint32_t *>(ctl.lut)[q] = reinterpret_cast<const uint32_t *>(g_cta_digit_lut.v)[q];
    const Camera cam = cams[view];
    const uint32_t bg = (uint32_t)S.bg[0] | ((uint32_t)S.bg[1] << 8) | ((uint32_t)S.bg[2] << 16);

    // ---------------------------------------------------------------- passes: the whole 32 x 32 tile (4 pixels per thread); if it does
    // not fit, its 16 x 16 quadrants, each split again into 8 x 8 when it does not fit (low
    // magnification: more light-field samples than output pixels under the tile); an 8 x 8 sub-tile that still does not fit
    // (strong minification) is rendered by 16 direct sample decodes per pixel
    int q = -1, r = -1;  // q < 0: whole tile; r < 0: 16 x 16 quadrant q; r = 0..3: its 8 x 8 quadrants
    while (q < 4) {
        const int ts = q < 0 ? kTile : (r < 0 ? 16 : 8);
        const int sx = q < 0 ? ox : ox + (q & 1) * 16 + (r < 0 ? 0 : (r & 1) * 8);
        const int sy = q < 0 ? oy : oy + (q >> 1) * 16 + (r < 0 ? 0 : (r >> 1) * 8);
        bool done = true;
        if (sx < W && sy < H) {
            PixTaps pt[kPPL];
            uint32_t rgb[kPPL];
#pragma unroll
            for (int p = 0; p < kPPL; ++p) rgb[p] = bg;
            PHASE_MARK(-1);
            setup_rays(S, cam, W, H, sx, sy, ts, pt);
            PHASE_MARK(0);
            PASS_STAT(ts == kTile ? 0 : ts == 16 ? 1 : 2);
            done = tile_pass<kArenaBytes>(S, ctl, arena, pt, rgb);
            if (done) PASS_STAT(ts == kTile ? 3 : ts == 16 ? 4 : 5);
            if (!done && r >= 0) {
                PASS_STAT(6);
                if (pt[0].uv != kNone) rgb[0] = direct_pixel(S, pt[0]);
                done = true;
            }
            if (done) {
                int x0, y, npix;
                thread_pixel(sx, sy, ts, x0, y, npix);
                if (q < 0) store4(out, view, W, H, x0, y, rgb, out_aligned);
                else store1(out, view, W, H, x0, y, npix > 0, rgb[0], out_aligned);
                PHASE_MARK(10);
            }
        }
        if (q < 0) q = done ? 4 : 0;
        else if (r < 0) { if (done) ++q; else r = 0; }
        else if (++r == 4) { r = -1; ++q; }
    }
}


// ---------------------------------------------------------------------------------------------------------------
// hmlfc_decode_views for B = 4 streams: one lane per block ROW segment (4 consecutive pixels of one block of one view).  The same
// per-row decode as phase B3 -- flag / rank record once per (level, channel), the row's 4 stored values from one pass over two
// 64-bit BISE windows, the motion record once, the motion-compensated reference row from at most two reference blocks -- without
// the shared-memory tables of the render kernel: whole views need no footprint.  PAPER.md:289-293; DESIGN.md section 3.
// kBlocks (hmlfc_decode_blocks): the segments are the 4 rows of arbitrary 4 x 4 blocks (u, v, bx, by) = blocks[g / 4] -- random access at
// the granularity the paper decodes at ("As a block of pixels are decoded ...") -- written as [n][4][4][3].
template <bool kBlocks>
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
        const int b = (t >> 2) * S.nbx + bx;
        const uint32_t g32 = (uint32_t)(b >> 5), bit = 1u << (b & 31), i0 = (uint32_t)((t & 3) << 2);
        for (int L = S.lmin; L < h; ++L) {
            const LevelDesc lv = S.lev[L];
            const int pu = u >> L, pv = v >> L;
            const uint32_t pc0 = lv.pc_base + (uint32_t)(pv * lv.UL + pu) * 3u;
            const uint32_t refpc0 = lv.pc_base + (uint32_t)((pv & ~1) * lv.UL + (pu & ~1)) * 3u;
            const bool predictive = ((pu | pv) & 1) != 0;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const uint4 d = ldg(S.pc + pc0 + c);
                const uint4 fr = ldg(S.flagrec + d.x + 4u * g32);
                uint2 own = make_uint2(0u, 0u);
                if (fr.x & bit) own = bise_row4(S.pay + d.y, ((fr.y + popc(fr.x & (bit - 1u))) << 4) + i0, d.w, lut);
                int e0 = (int)(int16_t)(own.x & 0xFFFFu), e1 = (int)own.x >> 16, e2 = (int)(int16_t)(own.y & 0xFFFFu), e3 = (int)own.y >> 16;
                if (predictive && (fr.z & bit)) {
                    const uint32_t mr = bise_at(S.mv + d.z, fr.w + popc(fr.z & (bit - 1u)), S.mv_layout, S.mv_m, lut);
                    int md, dx, dy;
                    mv_unpack(S, mr, md, dx, dy);
                    const int rx = s0 + dx, ry = t + dy;
                    if ((unsigned)ry < (unsigned)S.Ht) {
                        const uint4 dr = ldg(S.pc + refpc0 + c);
                        // the 4 reference samples (rx .. rx+3, ry) lie in the block row ry>>2, blocks rx>>2 and (rx>>2)+1
                        const int o = rx & 3, bxa = rx >> 2;
                        const uint32_t j0 = (uint32_t)((ry & 3) << 2);
                        const int rowb = (ry >> 2) * S.nbx;
                        uint2 qa = make_uint2(0u, 0u), qb = make_uint2(0u, 0u);
                        if ((unsigned)bxa < (unsigned)S.nbx) {
                            const int rb = rowb + bxa;
                            const uint4 rf = ldg(S.flagrec + dr.x + 4u * (uint32_t)(rb >> 5));
                            const uint32_t rbit = 1u << (rb & 31);
                            if (rf.x & rbit) qa = bise_row4(S.pay + dr.y, ((rf.y + popc(rf.x & (rbit - 1u))) << 4) + j0, dr.w, lut);
                        }
                        if (o && (unsigned)(bxa + 1) < (unsigned)S.nbx) {
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
                }
                a[c][0] += e0; a[c][1] += e1; a[c][2] += e2; a[c][3] += e3;
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
    decode_rows_kernel<false><<<(unsigned)blocks, kNT, 0, st>>>(S, reinterpret_cast<const int2 *>(d_views), n_seg, d_out, d_oob, aligned);
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
    decode_rows_kernel<true><<<(unsigned)blocks, kNT, 0, st>>>(S, reinterpret_cast<const int2 *>(d_blocks), n_seg, d_out, d_oob, aligned);
    if (n_launches) *n_launches += 1;
    return cudaGetLastError();
}

#ifdef HMLFC_PASS_STATS
extern "C" int hmlfc_debug_pass_stats(unsigned long long *out, int reset)
{
    cudaDeviceSynchronize();
    cudaMemcpyFromSymbol(out, g_pass_stats, sizeof(g_pass_stats));
    if (reset) { unsigned long long z[64] = {}; cudaMemcpyToSymbol(g_pass_stats, z, sizeof(z)); }
    return 0;
}
#endif

cudaError_t configure_render_cta()
{
    cudaError_t e = cudaFuncSetAttribute(render_cta_kernel<kArenaDefault, kMinBlocksDefault>, cudaFuncAttributeMaxDynamicSharedMemorySize, kArenaDefault);
    if (e != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(render_cta_kernel<kArenaSmall, kMinBlocksSmall>, cudaFuncAttributeMaxDynamicSharedMemorySize, kArenaSmall)) != cudaSuccess) return e;
    return cudaFuncSetAttribute(render_cta_kernel<kArenaBig, kMinBlocksBig>, cudaFuncAttributeMaxDynamicSharedMemorySize, kArenaBig);
}

cudaError_t launch_render_cta(const DevStream &S, const Camera *d_cams, int n_views, int W, int H, uint8_t *d_out, cudaStream_t st,
                              int *n_launches, int arena)
{
    if (n_views == 0) return cudaSuccess;
    if (S.B != 4) return cudaErrorInvalidValue;  // block-row tasks are written for 4 x 4 blocks; the caller dispatches other sizes elsewhere
    dim3 block(kNT), grid((unsigned)((W + kTile - 1) / kTile), (unsigned)((H + kTile - 1) / kTile), (unsigned)n_views);
    if (grid.y > 65535u) return cudaErrorInvalidValue;
    const int aligned = ((reinterpret_cast<uintptr_t>(d_out) & 3u) == 0 && (W % 4) == 0) ? 1 : 0;
    // measured, ms per step (68 KB x 3 / 104 KB x 2 / 50 KB x 4): cfg2 0.850 / 0.950 / 0.859, cfg3 0.975 / 0.837 / -, cfg3 with the eye on
    // the camera plane 2.24 / 1.08 / -, cfg4 1.010 / 1.163 / 1.035, cfg5 1.538 / 1.828 / 1.401, cfg1 0.070 / 0.039 / -
    if (arena < 0) arena = (long long)W * H < 2LL * S.Ws * S.Ht ? 1 : ((long long)W * H >= 8LL * S.Ws * S.Ht ? 2 : 0);
    const bool big = arena == 1;
    if (arena == 2) render_cta_kernel<kArenaSmall, kMinBlocksSmall><<<grid, block, kArenaSmall, st>>>(S, d_cams, W, H, d_out, aligned);
    else if (big) render_cta_kernel<kArenaBig, kMinBlocksBig><<<grid, block, kArenaBig, st>>>(S, d_cams, W, H, d_out, aligned);
    else render_cta_kernel<kArenaDefault, kMinBlocksDefault><<<grid, block, kArenaDefault, st>>>(S, d_cams, W, H, d_out, aligned);
    if (n_launches) *n_launches += 1;
    return cudaGetLastError();
}

}  // namespace hmlfc
