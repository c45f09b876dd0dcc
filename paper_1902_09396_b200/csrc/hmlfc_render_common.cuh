// Shared parts of the two fused decode + render kernels for B = 4 streams (sm_100a): hmlfc_render_tiles.cu (tile tables
// built by a kernel of their own, one pass per 32 x 32 tile -- the default) and hmlfc_render_cta.cu (tables built inside
// the CTA, quadtree of sub-tile passes -- every tile the first kernel hands over, and views at low magnification).
//
// PAPER.md:289-293 (decoding procedure), :309 (random access, "fast access to neighboring pixels for interpolation"),
// :73 / :409 (two-plane rendering).  Definitions: DESIGN.md sections 3 and 5.
//
// Vocabulary.  A tile's rays touch a (u,v) neighbourhood of at most 4 x 4 light-field VIEWS; view (iu, iv) has a footprint
// box of samples and owns one CELL per sample of that box (the float RGB patch the pixels finally gather from).  Under the
// views lie the SRV planes of every level ("SLOTS": a level-L plane is shared by the 2^L x 2^L views below it and is
// decoded ONCE per tile into an int16 accumulator of its own).
//   T   tables: view boxes and cells, slots and their boxes (build_tables);
//   B1  one lane per (slot, channel, block row of the slot's box): the row's flag/rank words are loaded once
//       (128-bit records), non-empty blocks are compacted into a record list;
//   B2  one lane per record: the block's motion record (BISE decode_at, once per block);
//   B3  one lane per (record, block row): the row's 4 stored values come from ONE pass over two 64-bit BISE
//       windows (plain / trit / quint without control flow); the motion-compensated reference row (two
//       neighbouring blocks of the reference SRV) likewise; written to the slot's int16 accumulator;
//   B4  one lane per cell: top-level RKV + the h per-level terms, inverse YCoCg-R, clamp -> float RGB patch (decode_patch);
//   C   every pixel gathers its 16 taps from the patch (128-bit loads) and blends with packed fp32 FMAs (blend_pixel).
// The footprint box PER VIEW needs no per-pixel work: every ray passes through the eye, so s is an affine function of u
// (and t of v) that depends on the camera alone (camera_affine); the pixels that touch view column a have u in
// [a-1, a+1) and hence s in the image of that interval (plus a rounding margin), intersected with the tile's box (axis_box).
#pragma once

#include "hmlfc_kernels.cuh"
#include "hmlfc_bise_row.cuh"

namespace hmlfc {

namespace {

constexpr int kPPL = 4;           // consecutive pixels per thread
constexpr int kMaxV = 4;          // views per axis of one tile's footprint
constexpr int kMaxViews = kMaxV * kMaxV;
constexpr int kMaxSlots = 40;     // 16 + 9 + 4 * 3 planes + slack (a pass with more planes is split)
constexpr int kMaxChunks = 512;   // 32-cell chunks of the patch
constexpr int kMinRec = 256;      // smallest record capacity worth starting with
constexpr uint32_t FULL = 0xffffffffu;
constexpr uint32_t kNone = 0xFFFFFFFFu;

// debug builds (-DHMLFC_PASS_STATS) count the passes of every size and why a pass was split
#ifdef HMLFC_PASS_STATS
__device__ unsigned long long g_pass_stats[64];  // [0..3] passes tried at quadtree level 0..3, [4..7] passes done, [8..] fail reasons, [16..] cycles of thread 0 per phase
__device__ long long g_phase_last[1 << 20];      // per CTA: clock of the previous mark
#define PASS_STAT(i) do { if (threadIdx.x == 0) atomicAdd(&g_pass_stats[i], 1ull); } while (0)
#define PHASE_MARK(i) do { if (threadIdx.x == 0) { const unsigned cta_ = (blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x; \
        const long long now_ = clock64(); if ((i) >= 0) atomicAdd(&g_pass_stats[16 + ((i) < 0 ? 0 : (i))], (unsigned long long)(now_ - g_phase_last[cta_ & ((1u << 20) - 1u)])); \
        g_phase_last[cta_ & ((1u << 20) - 1u)] = now_; } } while (0)
#else
#define PASS_STAT(i) do { } while (0)
#define PHASE_MARK(i) do { } while (0)
#endif

// n / d for n * d < 2^32 by one multiply-high (m == 0 encodes d <= 1)
__device__ __forceinline__ uint32_t magic_of(uint32_t d) { return d <= 1u ? 0u : 0xFFFFFFFFu / d + 1u; }
__device__ __forceinline__ uint32_t fdiv(uint32_t n, uint32_t m) { return m ? __umulhi(n, m) : n; }
// j / n for 0 <= j < 16, 1 <= n <= 4
__device__ __forceinline__ int div_small(int j, int n) { return n == 1 ? j : n == 2 ? (j >> 1) : n == 4 ? (j >> 2) : ((j * 11) >> 5); }

struct ViewInfo {   // view (iu, iv) of the tile's (u,v) neighbourhood, index iv * 4 + iu
    int s0, t0, ns, nt;          // footprint box of the view (ns == 0: no pixel of the tile touches it)
    int cellbase;                // first (view, sample) cell (a multiple of 32: a warp's cells belong to one view)
    uint32_t m_ns;               // magic multiplier of ns
    uint32_t rkv_lo, rkv_hi;     // index of the view's top-level RKV plane * Ht * Ws
};

struct SlotInfo {   // one SRV plane of one level under the tile's views (64 bytes)
    int s0, t0, ns, s1;          // sample box (union of the boxes of the views below); s1 = last column
    int t1, bx0, by0, nbw;       // last row; block box
    int accbase, nbh;            // first accumulator sample; block rows
    uint32_t pred;               // plane is predictive
    uint32_t pc0, refpc0;        // index of the plane's first descriptor / of its cluster's reference plane's
    int _pad[3];
};

struct TileHeader {  // 64 bytes
    int bu0, bv0, nu, nv;        // (u,v) range of the tile's taps
    int bs0, bs1, bt0, bt1;      // (s,t) box of all its taps
    int nslots, ncell, nacc, nbhmax;
    int status;                  // kTile*: what the tile's pass has to do
    uint32_t m_ps, m_nbh;        // magic multipliers of 3 * nbhmax and nbhmax (B1's item -> (slot, channel, block row))
    int _pad;
};
constexpr int kTileBackground = 0;  // no ray hits the slab
constexpr int kTileTables = 1;      // tables valid
constexpr int kTileGeneral = 2;     // left to the general kernel (irregular rays, too many views or planes)
constexpr int kTableHeadWords = (64 + 2 * kMaxV * 8 + kMaxViews * 32) / 16;  // 16-byte words of a TileTables before its slots

struct TileTables {  // what phase T produces
    TileHeader hdr;
    int2 colbox[kMaxV], rowbox[kMaxV];  // first / last sample column of the views of column iu, first / last row of those of row iv (first > last: none)
    ViewInfo view[kMaxViews];
    SlotInfo slot[kMaxSlots];
};

struct Ctl {
    int lo[4], hi[4];                    // (u0, v0) range of the tile's taps [0..1], (s, t) box of all its taps [2..3]
    float aff[2][4];                     // per axis: s = aff[0] + aff[1] u for every ray of this camera, rounding margin aff[2]
    Camera cam;
    TileTables tab;
    uint4 desc[kMaxSlots][3];            // descriptors of the slot's three plane-channels ...
    uint4 rdesc[kMaxSlots][3];           // ... and of its cluster's reference plane (predictive planes)
    int2 voff[kMaxViews][kMaxLevels];    // accumulator offset / row stride of the view's plane at level L
    int2 vcb[kMaxViews];                 // {cellbase - t0 * ns - s0, ns}: cell of sample (s,t) = x + t * y + s
    uint8_t chunkvw[kMaxChunks];         // view of the 32-cell chunk
    int n_rec;
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
__device__ __forceinline__ uint32_t blend16(float fu, float fv, float fs, float ft, Fetch fetch)
{
    const float ws0 = 1.0f - fs, wt0 = 1.0f - ft, wu0 = 1.0f - fu, wv0 = 1.0f - fv;
    const float wst[4] = {ws0 * wt0, fs * wt0, ws0 * ft, fs * ft};
    const float wuv[4] = {wu0 * wv0, fu * wv0, wu0 * fv, fu * fv};
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

// a pixel whose taps are not in the tile's patch: 16 direct sample decodes (the unshared definition)
__device__ __noinline__ uint32_t direct_pixel(const DevStream &S, const PixTaps k)
{
    const int u0 = k.uv & 0xFFF, v0 = (k.uv >> 12) & 0xFFF, s0 = k.st & 0x3FFF, t0 = (k.st >> 14) & 0x3FFF;
    const int u1 = u0 + (int)((k.uv >> 24) & 1u), v1 = v0 + (int)((k.uv >> 25) & 1u);
    const int s1 = s0 + (int)((k.st >> 28) & 1u), t1 = t0 + (int)((k.st >> 29) & 1u);
    uint32_t c8[16];
#pragma unroll 1
    for (int a = 0; a < 16; ++a) c8[a] = decode_rgb8(S, (a & 4) ? u1 : u0, (a & 8) ? v1 : v0, (a & 1) ? s1 : s0, (a & 2) ? t1 : t0);
    return blend16(k.fu, k.fv, k.fs, k.ft, [&](int a, int b) {
        const uint32_t c = c8[a * 4 + b];
        return make_float4((float)(c & 0xFFu), (float)((c >> 8) & 0xFFu), (float)((c >> 16) & 0xFFu), 0.f);
    });
}

__device__ __forceinline__ PixTaps pack_taps(const Taps &k)
{
    PixTaps t;
    t.uv = (uint32_t)k.u0 | ((uint32_t)k.v0 << 12) | ((uint32_t)(k.u1 - k.u0) << 24) | ((uint32_t)(k.v1 - k.v0) << 25);
    t.st = (uint32_t)k.s0 | ((uint32_t)k.t0 << 14) | ((uint32_t)(k.s1 - k.s0) << 28) | ((uint32_t)(k.t1 - k.t0) << 29);
    t.fu = k.fu; t.fv = k.fv; t.fs = k.fs; t.ft = k.ft;
    return t;
}

// 16-tap footprint of the pixel with screen coordinates (px, py)
__device__ __forceinline__ PixTaps pixel_taps(const DevStream &S, const Camera &cam, float px, float py, bool inside)
{
    PixTaps t;
    t.uv = kNone; t.st = 0u;
    t.fu = t.fv = t.fs = t.ft = 0.f;
    if (inside) {
        const Ray r = ray_from_screen(S, cam, px, py);
        if (r.hit) {
            const Taps k = tap_setup(S, r);
            t = pack_taps(k);
        }
    }
    return t;
}

// C for one pixel: its 16 taps from the patch, blended.  kGuard: a tap outside its view's box (the tables came from a
// conservative estimate of the tile's footprint, hmlfc_render_tiles.cu) sends the pixel to the direct decode instead.
template <bool kGuard>
__device__ __forceinline__ uint32_t blend_taps(const DevStream &S, const Ctl &ctl, const float4 *__restrict__ patch, const Taps &k, int bu0, int bv0)
{
    const int iu = k.u0 - bu0, iv = k.v0 - bv0;
    const int s0 = k.s0, t0 = k.t0;
    const int du = k.u1 - k.u0, dv = (k.v1 - k.v0) << 2;
    const int ds = k.s1 - k.s0, dt = k.t1 - k.t0;
    const int vw0 = iv * 4 + iu;
    if (kGuard) {
        // a view's box is (its column's sample columns) x (its row's sample rows): two interval tests per axis cover the four views
        bool ok = iu >= 0 && iv >= 0 && iu + du < kMaxV && iv * 4 + dv < kMaxViews;
        if (ok) {
            const int2 c0 = ctl.tab.colbox[iu], c1 = ctl.tab.colbox[iu + du], r0 = ctl.tab.rowbox[iv], r1 = ctl.tab.rowbox[iv + (dv >> 2)];
            ok = s0 >= max(c0.x, c1.x) && s0 + ds <= min(c0.y, c1.y) && t0 >= max(r0.x, r1.x) && t0 + dt <= min(r0.y, r1.y);
        }
        if (!ok) {
#ifdef HMLFC_PASS_STATS
            atomicAdd(&g_pass_stats[12], 1ull);
#endif
            return direct_pixel(S, pack_taps(k));
        }
    }
    int vb[4], vs[4];
#pragma unroll
    for (int a = 0; a < 4; ++a) {
        const int2 cb = ctl.vcb[vw0 + ((a & 1) ? du : 0) + ((a & 2) ? dv : 0)];
#ifdef HMLFC_BOX_CHECK
        {
            const ViewInfo &vi = ctl.tab.view[vw0 + ((a & 1) ? du : 0) + ((a & 2) ? dv : 0)];
            if (s0 < vi.s0 || s0 + ds >= vi.s0 + vi.ns || t0 < vi.t0 || t0 + dt >= vi.t0 + vi.nt) atomicAdd(&g_pass_stats[12], 1ull);
        }
#endif
        vb[a] = cb.x + t0 * cb.y + s0;
        vs[a] = dt ? cb.y : 0;
    }
    return blend16(k.fu, k.fv, k.fs, k.ft, [&](int a, int b) { return patch[vb[a] + ((b & 1) ? ds : 0) + ((b & 2) ? vs[a] : 0)]; });
}

__device__ __forceinline__ uint32_t blend_pixel(const DevStream &S, const Ctl &ctl, const float4 *__restrict__ patch, const PixTaps k, int bu0, int bv0)
{
    Taps t;
    t.u0 = (int)(k.uv & 0xFFF); t.v0 = (int)((k.uv >> 12) & 0xFFF); t.s0 = (int)(k.st & 0x3FFF); t.t0 = (int)((k.st >> 14) & 0x3FFF);
    t.u1 = t.u0 + (int)((k.uv >> 24) & 1u); t.v1 = t.v0 + (int)((k.uv >> 25) & 1u);
    t.s1 = t.s0 + (int)((k.st >> 28) & 1u); t.t1 = t.t0 + (int)((k.st >> 29) & 1u);
    t.fu = k.fu; t.fv = k.fv; t.fs = k.fs; t.ft = k.ft;
    return blend_taps<false>(S, ctl, patch, t, bu0, bv0);
}

// Footprint interval along one axis of the views / planes that cover grid positions [a0, a1] of that axis: the pixels that touch
// them have a continuous grid coordinate in [a0 - 1, a1 + 1) and, every ray passing through the eye, an image-plane coordinate
// of aff[0] + aff[1] * (grid coordinate) up to the rounding margin aff[2]; taps are floor(.) and floor(.) + 1.  Clipped to the tile's
// own box [lo, hi].  A degenerate camera (eye on the camera plane: all pixels share one grid coordinate) has a non-finite map
// and gets the tile's box.
__device__ __forceinline__ void axis_box(const float (&aff)[4], int a0, int a1, int lo, int hi, int &b0, int &b1)
{
    const float e0 = fmaf(aff[1], (float)(a0 - 1), aff[0]), e1 = fmaf(aff[1], (float)(a1 + 1), aff[0]);
    const float x0 = fminf(e0, e1) - aff[2], x1 = fmaxf(e0, e1) + aff[2];
    b0 = lo; b1 = hi;
    if (x0 > (float)lo && x0 < 1e9f) b0 = (int)floorf(x0);          // NaN / infinities fail the comparisons: tile box
    if (x1 < (float)hi && x1 > -1e9f) b1 = (int)floorf(x1) + 1;
    b0 = max(b0, lo); b1 = min(b1, hi);
}

// s = aff[0] + aff[1] * u (index units) for every ray of the camera along one axis, and the margin aff[2] of that relation between
// the fp32 values the ray set-up computes.  u_w = e + l0 D, s_w = e + l1 D with l0 = (0 - ez) / Dz, l1 = (z_st - ez) / Dz, so
// s_w - e = k (u_w - e) with k = (z_st - ez) / (0 - ez) whatever D is.  The margin covers the dozen roundings of either chain (64 ulps of
// the magnitudes involved) and the fp32 evaluation of aff[0] + aff[1] * u itself; a box that is a sample too wide costs a few decodes,
// one that is too narrow would be wrong.
__device__ __forceinline__ void camera_affine(const DevStream &S, const Camera &cam, int axis, float (&aff)[4])
{
    const float e = cam.eye[axis], ez = cam.eye[2];
    const float uo = S.uv_origin[axis], us = S.uv_step[axis], so = S.st_origin[axis], ss = S.st_step[axis];
    const float k = (S.z_st - ez) / (0.0f - ez), rs = 1.0f / ss;
    const float beta = k * us * rs;
    const float n_uv = (float)(axis == 0 ? S.U : S.V), n_st = (float)(axis == 0 ? S.Ws : S.Ht);
    const float mw = fmaxf(fmaxf(fabsf(e), fabsf(uo) + fabsf(us) * n_uv), fmaxf(fabsf(so) + fabsf(ss) * n_st, 1.0f));
    const float mag = (fabsf(e - so) + fabsf(k) * fabsf(uo - e)) * fabsf(rs) + fabsf(beta) * (n_uv + 2.0f);  // terms of aff[0] + aff[1] u
    aff[0] = ((e - so) + k * (uo - e)) * rs;
    aff[1] = beta;
    aff[2] = 64.0f * 5.9604644775390625e-8f * (n_st + mw * fabsf(rs) + fabsf(beta) * (n_uv + mw / fabsf(us)) + mag) + 1e-5f;
    aff[3] = 0.0f;
}

// planes of level L over the views [bu0, bu0 + nu) x [bv0, bv0 + nv): a (nuL x nvL) rectangle starting at (bu0 >> L, bv0 >> L)
__device__ __forceinline__ int level_nu(int b0, int n, int L) { return ((b0 + n - 1) >> L) - (b0 >> L) + 1; }

// ---------------------------------------------------------------------------------------------------------------
// T, view half (one warp, all 32 lanes call): boxes and cells of the views of the ranges rg (bu0 .. bt1); writes tab.view[], the
// ranges and ncell of tab.hdr.
__device__ __forceinline__ void build_view_table(const DevStream &S, const float (&aff)[2][4], const TileHeader rg, TileTables &tab)
{
    const int lane = threadIdx.x & 31, h = S.h;
    const int bu0 = rg.bu0, bv0 = rg.bv0, nu = rg.nu, nv = rg.nv;
    const int iu = lane & 3, iv = (lane >> 2) & 3;
    int vs0 = 0, vt0 = 0, vns = 0, vnt = 0;
    int a0 = 1, a1 = 0, c0 = 1, c1 = 0;
    if (lane < kMaxViews && iu < nu && iv < nv) {
        axis_box(aff[0], bu0 + iu, bu0 + iu, rg.bs0, rg.bs1, a0, a1);
        axis_box(aff[1], bv0 + iv, bv0 + iv, rg.bt0, rg.bt1, c0, c1);
        if (a0 <= a1 && c0 <= c1) { vs0 = a0; vt0 = c0; vns = a1 - a0 + 1; vnt = c1 - c0 + 1; }
    }
    if (lane < kMaxV) tab.colbox[lane] = (iu < nu && a0 <= a1) ? make_int2(a0, a1) : make_int2(1, 0);                 // lanes (iu, 0)
    if (lane < kMaxViews && iu == 0) tab.rowbox[iv] = (iv < nv && c0 <= c1) ? make_int2(c0, c1) : make_int2(1, 0);    // lanes (0, iv)
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
        vi.m_ns = magic_of((uint32_t)vns);
        const unsigned long long ro = (unsigned long long)(((bv0 + iv) >> h) * S.UH + ((bu0 + iu) >> h)) *
                                      (unsigned long long)S.Ht * (unsigned long long)S.Ws;
        vi.rkv_lo = (uint32_t)ro; vi.rkv_hi = (uint32_t)(ro >> 32);
        tab.view[lane] = vi;
    }
    if (lane == 0) {
        tab.hdr.bu0 = bu0; tab.hdr.bv0 = bv0; tab.hdr.nu = nu; tab.hdr.nv = nv;
        tab.hdr.bs0 = rg.bs0; tab.hdr.bs1 = rg.bs1; tab.hdr.bt0 = rg.bt0; tab.hdr.bt1 = rg.bt1;
        tab.hdr.ncell = ncell;
    }
}

// T, plane half (one warp, all 32 lanes call): the SRV planes of every level under the views; writes tab.slot[], hdr.nslots / nacc / nbhmax.
__device__ __forceinline__ void build_slot_table(const DevStream &S, const float (&aff)[2][4], const TileHeader rg, TileTables &tab)
{
    const int lane = threadIdx.x & 31, h = S.h;
    const int bu0 = rg.bu0, bv0 = rg.bv0, nu = rg.nu, nv = rg.nv;
    const int bs0 = rg.bs0, bs1 = rg.bs1, bt0 = rg.bt0, bt1 = rg.bt1;
    // lane L owns level L: planes of the level, then the running count over the levels (progressive decoding: none below lmin)
    const int cntL = (lane >= S.lmin && lane < h) ? level_nu(bu0, nu, lane) * level_nu(bv0, nv, lane) : 0;
    int lincl = cntL;
#pragma unroll
    for (int o = 1; o < kMaxLevels; o <<= 1) {
        const int n = __shfl_up_sync(FULL, lincl, o);
        if (lane >= o) lincl += n;
    }
    const int nslots = __shfl_sync(FULL, lincl, kMaxLevels - 1);
    int accrun = 0, nbhmax = 0;
    if (nslots <= kMaxSlots) {
        for (int sb = 0; sb < nslots; sb += 32) {
            const int s = sb + lane;
            int L = 0, base = 0;
            for (int l = 0; l < h - 1; ++l) {  // level of slot s: the last one whose first slot is <= s
                const int end = __shfl_sync(FULL, lincl, l);
                if (s >= end) { L = l + 1; base = end; }
            }
            SlotInfo si;
            si.pred = 0u; si.pc0 = si.refpc0 = 0u; si._pad[0] = si._pad[1] = si._pad[2] = 0;
            si.s0 = si.t0 = 0; si.ns = 0; si.s1 = si.t1 = -1; si.bx0 = si.by0 = 0; si.nbw = 0; si.nbh = 0;
            int nsamp = 0;
            if (s < nslots) {
                const int n = level_nu(bu0, nu, L);
                const int jj = s - base, jv = div_small(jj, n);
                const int pv = (bv0 >> L) + jv, pu = (bu0 >> L) + (jj - jv * n);
                const LevelDesc lv = S.lev[L];
                si.pc0 = lv.pc_base + (uint32_t)(pv * lv.UL + pu) * 3u;
                si.refpc0 = lv.pc_base + (uint32_t)((pv & ~1) * lv.UL + (pu & ~1)) * 3u;
                si.pred = (uint32_t)((pu | pv) & 1);
                // box of the views below this plane
                int a0, a1, c0, c1;
                axis_box(aff[0], max(pu << L, bu0), min(((pu + 1) << L) - 1, bu0 + nu - 1), bs0, bs1, a0, a1);
                axis_box(aff[1], max(pv << L, bv0), min(((pv + 1) << L) - 1, bv0 + nv - 1), bt0, bt1, c0, c1);
                if (a0 <= a1 && c0 <= c1) {
                    si.s0 = a0; si.t0 = c0; si.s1 = a1; si.t1 = c1; si.ns = a1 - a0 + 1;
                    si.bx0 = a0 >> 2; si.by0 = c0 >> 2;
                    si.nbw = (a1 >> 2) - si.bx0 + 1; si.nbh = (c1 >> 2) - si.by0 + 1;
                    nsamp = si.ns * (c1 - c0 + 1);
                }
            }
            int ai = nsamp;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int n1 = __shfl_up_sync(FULL, ai, o);
                if (lane >= o) ai += n1;
            }
            si.accbase = accrun + ai - nsamp;
            if (s < nslots) tab.slot[s] = si;
            accrun += __shfl_sync(FULL, ai, 31);
            nbhmax = max(nbhmax, __reduce_max_sync(FULL, si.nbh));
        }
    }
    if (lane == 0) {
        tab.hdr.nslots = nslots; tab.hdr.nacc = accrun; tab.hdr.nbhmax = nbhmax;
        tab.hdr.m_ps = magic_of((uint32_t)(3 * nbhmax)); tab.hdr.m_nbh = magic_of((uint32_t)nbhmax);
    }
}

// do the tables fit an arena of kArenaBytes?  accumulators (8 bytes per slot sample), then the patch (16 bytes per cell) aliased by
// the record list (32 bytes each)
template <int kArenaBytes>
__device__ __forceinline__ bool tables_fit(const TileHeader &hd)
{
    const long long rest = (long long)kArenaBytes - (((long long)hd.nacc * 8 + 15) & ~15LL);
    return hd.nslots <= kMaxSlots && hd.ncell <= 32 * kMaxChunks && rest >= (long long)hd.ncell * 16 && rest >= (long long)kMinRec * 32;
}

// ---------------------------------------------------------------------------------------------------------------
// Phases B1-B4 for the tile whose tables are in ctl.tab (visible to all threads; they fit the arena): the float RGB patch of every
// (view, sample) cell.  kZeroFrom: the first 16-byte word of the accumulator region this function still has to zero (the caller zeroed
// the words before it and ctl.n_rec).  Returns false (CTA-uniform) when the record list does not fit; ends with a barrier either way.
// kCs: chroma-subsampled streams (R18): the Co / Cg plane-channels have their own (half-resolution) block grid in B1 - B3; the
// accumulators stay at luma resolution (a chroma sample is written to the up to 2 x 2 cells it covers), so B4 and the tables do not change.
template <int kArenaBytes, int kNT, bool kSubpel = false, bool kCs = false>
__device__ __forceinline__ bool decode_patch(const DevStream &S, Ctl &ctl, unsigned char *__restrict__ arena, int zero_from)
{
    const int tid = threadIdx.x, lane = tid & 31;
    const int h = S.h;
    const TileHeader hd = ctl.tab.hdr;
    const int ncell = hd.ncell, nacc = hd.nacc, nslots = hd.nslots, nbhmax = hd.nbhmax;
    const int bu0 = hd.bu0, bv0 = hd.bv0, nu = hd.nu, nv = hd.nv;
    const long long rest = (long long)kArenaBytes - (((long long)nacc * 8 + 15) & ~15LL);
    const int reccap = (int)min(rest / 32, 0x7fffffLL);
    uint2 *acc = reinterpret_cast<uint2 *>(arena);
    unsigned char *region2 = arena + (((size_t)nacc * 8 + 15) & ~(size_t)15);
    uint4 *rec = reinterpret_cast<uint4 *>(region2);      // [reccap][2]
    float4 *patch = reinterpret_cast<float4 *>(region2);  // [ncell], after the records are dead
    // ---------------------------------------------------- zero the accumulators; per-view cell offsets, chunk -> view, accumulator
    // offsets of every (view, level); the planes' descriptors (and their reference planes') go to shared memory for B2 and B3
    static_assert(6 * kMaxSlots <= 256 && kNT >= 256, "one descriptor per thread");
    uint4 dsc = make_uint4(0u, 0u, 0u, 0u);
    {
        uint4 *z = reinterpret_cast<uint4 *>(arena);
        const int nz = (nacc + 1) >> 1;
        for (int q = zero_from + tid; q < nz; q += kNT) z[q] = make_uint4(0u, 0u, 0u, 0u);
        if (tid < nslots * 6) {  // loaded now, stored behind B1 (6 * kMaxSlots <= 256 threads): B1 does not wait for them
            const uint32_t s = fdiv((uint32_t)tid, 0x2AAAAAABu), j = (uint32_t)tid - 6u * s;  // tid / 6
            const SlotInfo &sl = ctl.tab.slot[s];
            dsc = ldg(S.pc + (j < 3u ? sl.pc0 + j : sl.refpc0 + (j - 3u)));
        }
        for (int q = tid; q < kMaxViews * h; q += kNT) {
            const int L = q >> 4, vw = q & 15;
            const ViewInfo &vi = ctl.tab.view[vw];
            if (L < S.lmin || vi.ns == 0) continue;
            const int iu = vw & 3, iv = vw >> 2;
            int base = 0;
            for (int l = S.lmin; l < L; ++l) base += level_nu(bu0, nu, l) * level_nu(bv0, nv, l);
            const int sidx = base + (((bv0 + iv) >> L) - (bv0 >> L)) * level_nu(bu0, nu, L) + (((bu0 + iu) >> L) - (bu0 >> L));
            const SlotInfo &sl = ctl.tab.slot[sidx];
            ctl.voff[vw][L] = make_int2(sl.accbase + (vi.t0 - sl.t0) * sl.ns + (vi.s0 - sl.s0), sl.ns);
        }
        if (tid >= kNT - kMaxViews) {
            const int vw = tid - (kNT - kMaxViews);
            const ViewInfo &vi = ctl.tab.view[vw];
            ctl.vcb[vw] = make_int2(vi.cellbase - vi.t0 * vi.ns - vi.s0, vi.ns);
            const int c1 = min((vi.cellbase + ((vi.ns * vi.nt + 31) & ~31)) >> 5, kMaxChunks);
            for (int c = vi.cellbase >> 5; c < c1; ++c) ctl.chunkvw[c] = (uint8_t)vw;
        }
    }
    // ---------------------------------------------------- B1: one lane per (slot, channel, block row): flag words -> records
    {
        const int per_slot = 3 * nbhmax, nitems = nslots * per_slot;
        const uint32_t m_ps = hd.m_ps, m_nbh = hd.m_nbh;
        for (int base = 0; base < nitems; base += kNT) {
            const int it = base + tid;
            bool on = it < nitems;
            uint32_t pred = 0u, sc = 0u;
            size_t frbase = 0;
            int b0 = 0, b1 = -1, by = 0, rowb = 0;
            if (on) {
                const uint32_t s = fdiv((uint32_t)it, m_ps), r = (uint32_t)it - s * (uint32_t)per_slot;
                const uint32_t c = fdiv(r, m_nbh), jr = r - c * (uint32_t)nbhmax;
                const SlotInfo &sl = ctl.tab.slot[s];
                // the channel's block box: the slot's, or (kCs, chroma) the blocks of the half-resolution plane under the slot's sample box
                int cbx0 = sl.bx0, cby0 = sl.by0, cnbw = sl.nbw, cnbh = sl.nbh, cnbx = S.nbx;
                if (kCs && c > 0u) {
                    cbx0 = sl.s0 >> 3; cby0 = sl.t0 >> 3; cnbw = (sl.s1 >> 3) - cbx0 + 1; cnbh = (sl.t1 >> 3) - cby0 + 1; cnbx = S.nbx_c;
                    if (sl.ns == 0) cnbh = 0;
                }
                on = (int)jr < cnbh;
                if (on) {
                    frbase = flag_index(S, sl.pc0 + c, 0u);  // = the descriptor's flag record base, without waiting for it
                    sc = s | (c << 6);
                    pred = sl.pred;
                    by = cby0 + (int)jr;
                    rowb = by * cnbx;
                    b0 = rowb + cbx0; b1 = b0 + cnbw - 1;
                }
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
                    // rank of the block's payload * 16, rank of its motion record, slot | channel | block row | block column
                    if (idx < reccap)
                        rec[2 * idx] = make_uint4(hr ? ((fr.y + popc(fr.x & (bit - 1u))) << 4) : kNone, hp ? (fr.w + popc(fr.z & (bit - 1u))) : kNone,
                                              sc | ((uint32_t)by << 8) | ((uint32_t)((g << 5) + bp - rowb) << 20), 0u);
                    ++idx;
                }
            }
        }
    }
    if (tid < nslots * 6) {
        const uint32_t s = fdiv((uint32_t)tid, 0x2AAAAAABu), j = (uint32_t)tid - 6u * s;
        if (j < 3u) ctl.desc[s][j] = dsc; else ctl.rdesc[s][j - 3u] = dsc;
    }
    __syncthreads();
    PHASE_MARK(5);
    const int nrec = ctl.n_rec;
    if (nrec > reccap) {
        PASS_STAT(11);
        __syncthreads();  // every thread has read the record count (the caller resets it)
        return false;
    }
    // ------------------------------------------------ B2: one lane per record of a predicted block: its motion record (BISE decode_at), then
    // the flag / rank words of the (up to 2 x 2) reference blocks its four re-compensated rows read from -> second half of the record,
    // {significant | rank * 16} per reference block.  B3's loads then depend on nothing but the record: one round trip per task.
    for (int rr = tid; rr < nrec; rr += kNT) {
        const uint4 r0 = rec[2 * rr];
        if (r0.y == kNone) continue;
        const uint32_t s = r0.z & 63u, c = (r0.z >> 6) & 3u;
        int md, dx, dy;
        mv_unpack(S, bise_at(S.mv + ctl.desc[s][c].z, r0.y, S.mv_layout, S.mv_m, ctl.lut), md, dx, dy);
        const uint4 dr = ctl.rdesc[s][c];
        // first reference sample of the block; kSubpel (R28): the offsets count half pixels, a reference value is the mean of the
        // 1 / 2 / 4 samples from (rx, ry0) on, so a block reads one more column (fx) and one more row (fy)
        const int fx = kSubpel ? (dx & 1) : 0, fy = kSubpel ? (dy & 1) : 0;
        const int rx = (int)((r0.z >> 20) << 2) + (kSubpel ? (dx >> 1) : dx), ry0 = (int)(((r0.z >> 8) & 0xFFFu) << 2) + (kSubpel ? (dy >> 1) : dy);
        const int bxa = rx >> 2, bya = ry0 >> 2;  // arithmetic shifts: floor for positions left of / above the image
        const int cnbx = (kCs && c > 0u) ? S.nbx_c : S.nbx, cnby = (kCs && c > 0u) ? S.nby_c : S.nby;  // the channel's block grid
        uint32_t e[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int bx = bxa + (j & 1), by = bya + (j >> 1);
            e[j] = 0u;
            // needed at all: the second column only if the row straddles two blocks, the second block row likewise
            if ((unsigned)bx < (unsigned)cnbx && (unsigned)by < (unsigned)cnby && (!(j & 1) || (rx & 3) || fx) && (!(j >> 1) || (ry0 & 3) || fy)) {
                const int b = by * cnbx + bx;
                const uint2 fr = __ldg(reinterpret_cast<const uint2 *>(S.flagrec + dr.x + 4u * (uint32_t)(b >> 5)));  // {res bits, res rank}
                const uint32_t bit = 1u << (b & 31);
                if (fr.x & bit) e[j] = ((fr.y + popc(fr.x & (bit - 1u))) << 4) | 1u;
            }
        }
        rec[2 * rr].y = ((uint32_t)md << 16) | ((uint32_t)(dx + S.mv_off) << 8) | (uint32_t)(dy + S.mv_off);  // (mv_off <= 127: the caller's condition)
        rec[2 * rr + 1] = make_uint4(e[0], e[1], e[2], e[3]);
    }
    __syncthreads();
    PHASE_MARK(6);
    // ------------------------------------------------ B3: one lane per (record, block row): 4 stored / re-compensated values (neighbouring
    // lanes work on neighbouring blocks of one plane: their payload words share sectors and they take the same branches)
    {
        int16_t *acc16 = reinterpret_cast<int16_t *>(arena);
        for (int t = tid; t < 4 * nrec; t += kNT) {
            const int rr = t >> 2, ky = t & 3;
            const uint4 r0 = rec[2 * rr];
            const uint32_t s = r0.z & 63u, c = (r0.z >> 6) & 3u;
            const SlotInfo &sl = ctl.tab.slot[s];
            const int yy0 = (int)(((r0.z >> 8) & 0xFFFu) << 2), yy = yy0 + ky;
            const int st0 = sl.t0, st1 = sl.t1;
            const int csh = (kCs && c > 0u) ? 1 : 0;  // the channel's samples are (s >> csh, t >> csh); its image has Ht >> csh rows
            if (yy < (st0 >> csh) || yy > (st1 >> csh)) continue;
            const int cHt = S.Ht >> csh;
            const int xx = (int)((r0.z >> 20) << 2);
            const uint4 d = ctl.desc[s][c];
            uint2 own = make_uint2(0u, 0u);
            if (r0.x != kNone) own = bise_row4(S.pay + d.y, r0.x + (uint32_t)(ky << 2), d.w, ctl.lut);
            int e0 = (int)(int16_t)(own.x & 0xFFFFu), e1 = (int)own.x >> 16, e2 = (int)(int16_t)(own.y & 0xFFFFu), e3 = (int)own.y >> 16;
            if (r0.y != kNone) {
                const int md = (int)((r0.y >> 16) & 1u), dx = (int)((r0.y >> 8) & 0xFFu) - S.mv_off, dy = (int)(r0.y & 0xFFu) - S.mv_off;
                const uint4 dr = ctl.rdesc[s][c];
                const uint4 re = rec[2 * rr + 1];
                if (!kSubpel) {
                    const int rx = xx + dx, ry = yy + dy;
                    if ((unsigned)ry < (unsigned)cHt) {
                        // the 4 reference samples (rx .. rx+3, ry) lie in the block row ry>>2, blocks rx>>2 and (rx>>2)+1: B2 looked them up
                        const int o = rx & 3;
                        const bool second_row = (ry >> 2) != ((yy0 + dy) >> 2);
                        const uint32_t ea = second_row ? re.z : re.x, eb = second_row ? re.w : re.y;
                        const uint32_t i0 = (uint32_t)((ry & 3) << 2);
                        uint2 qa = make_uint2(0u, 0u), qb = make_uint2(0u, 0u);
                        if (ea & 1u) qa = bise_row4(S.pay + dr.y, (ea & ~15u) + i0, dr.w, ctl.lut);
                        if (eb & 1u) qb = bise_row4(S.pay + dr.y, (eb & ~15u) + i0, dr.w, ctl.lut);
                        // samples o .. o+3 of the 8-sample string qa | qb
                        uint32_t w0 = qa.x, w1 = qa.y, w2 = qb.x, w3 = qb.y;
                        if (o & 2) { w0 = w1; w1 = w2; w2 = w3; }
                        const uint32_t sh = (uint32_t)(o & 1) << 4;
                        const uint32_t q01 = __funnelshift_r(w0, w1, sh), q23 = __funnelshift_r(w1, w2, sh);
                        const int q0 = (int)(int16_t)(q01 & 0xFFFFu), q1 = (int)q01 >> 16, q2 = (int)(int16_t)(q23 & 0xFFFFu), q3 = (int)q23 >> 16;
                        // R10: subtractive P = e + R, additive P = e - R
                        if (md) { e0 -= q0; e1 -= q1; e2 -= q2; e3 -= q3; }
                        else { e0 += q0; e1 += q1; e2 += q2; e3 += q3; }
                    }
                } else {
                    // half-pel (R28): samples (rx .. rx+3+fx) of the rows ry and, if fy, ry + 1, summed and rounded half up; a row outside
                    // the image and a sample in an insignificant block contribute 0 to the sum
                    const int fx = dx & 1, fy = dy & 1;
                    const int rx = xx + (dx >> 1), ry = yy + (dy >> 1), o = rx & 3, bya = (yy0 + (dy >> 1)) >> 2;
                    int h0 = 0, h1 = 0, h2 = 0, h3 = 0;
#pragma unroll
                    for (int jr = 0; jr < 2; ++jr) {
                        const int r = ry + jr;
                        if ((jr && !fy) || (unsigned)r >= (unsigned)cHt) continue;
                        const bool second_row = (r >> 2) != bya;
                        const uint32_t ea = second_row ? re.z : re.x, eb = second_row ? re.w : re.y;
                        const uint32_t i0 = (uint32_t)((r & 3) << 2);
                        uint2 qa = make_uint2(0u, 0u), qb = make_uint2(0u, 0u);
                        if (ea & 1u) qa = bise_row4(S.pay + dr.y, (ea & ~15u) + i0, dr.w, ctl.lut);
                        if (eb & 1u) qb = bise_row4(S.pay + dr.y, (eb & ~15u) + i0, dr.w, ctl.lut);
                        // samples o .. o+4 of the 8-sample string qa | qb (o + 4 <= 7)
                        uint32_t w0 = qa.x, w1 = qa.y, w2 = qb.x, w3 = qb.y;
                        if (o & 2) { w0 = w1; w1 = w2; w2 = w3; w3 = 0u; }
                        const uint32_t sh = (uint32_t)(o & 1) << 4;
                        const uint32_t q01 = __funnelshift_r(w0, w1, sh), q23 = __funnelshift_r(w1, w2, sh), q45 = __funnelshift_r(w2, w3, sh);
                        const int q0 = (int)(int16_t)(q01 & 0xFFFFu), q1 = (int)q01 >> 16, q2 = (int)(int16_t)(q23 & 0xFFFFu), q3 = (int)q23 >> 16;
                        const int q4 = (int)(int16_t)(q45 & 0xFFFFu);
                        h0 += q0 + (fx ? q1 : 0); h1 += q1 + (fx ? q2 : 0); h2 += q2 + (fx ? q3 : 0); h3 += q3 + (fx ? q4 : 0);
                    }
                    const int k = fx + fy;  // log2 of the number of samples; the rounding term n / 2 = 0, 1, 2 = k
                    const int q0 = (h0 + k) >> k, q1 = (h1 + k) >> k, q2 = (h2 + k) >> k, q3 = (h3 + k) >> k;
                    if (md) { e0 -= q0; e1 -= q1; e2 -= q2; e3 -= q3; }
                    else { e0 += q0; e1 += q1; e2 += q2; e3 += q3; }
                }
            }
            const int ss0 = sl.s0, ss1 = sl.s1;
            if (!csh) {
                int16_t *dst = acc16 + (((sl.accbase + (yy - st0) * sl.ns + (xx - sl.s0)) << 2) + (int)c);
                if (xx >= ss0 && xx <= ss1) dst[0] = (int16_t)e0;
                if (xx + 1 >= ss0 && xx + 1 <= ss1) dst[4] = (int16_t)e1;
                if (xx + 2 >= ss0 && xx + 2 <= ss1) dst[8] = (int16_t)e2;
                if (xx + 3 >= ss0 && xx + 3 <= ss1) dst[12] = (int16_t)e3;
            } else {
                // a chroma sample (x, y) is the value of the luma-resolution cells (2x .. 2x+1, 2y .. 2y+1) (R18: nearest-neighbour replication)
                const int ev[4] = {e0, e1, e2, e3};
#pragma unroll
                for (int jy = 0; jy < 2; ++jy) {
                    const int ly = 2 * yy + jy;
                    if (ly < st0 || ly > st1) continue;
                    int16_t *row = acc16 + (((sl.accbase + (ly - st0) * sl.ns - ss0) << 2) + (int)c);
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const int lx = 2 * xx + i;
                        if (lx >= ss0 && lx <= ss1) row[lx << 2] = (int16_t)ev[i >> 1];
                    }
                }
            }
        }
    }
    __syncthreads();
    PHASE_MARK(7);
    // ------------------------------------------------ B4: top-level RKV + per-level terms -> float RGB patch
    for (int q = tid; q < ncell; q += kNT) {
        const int vw = ctl.chunkvw[q >> 5];
        const ViewInfo vi = ctl.tab.view[vw];
        const uint32_t local = (uint32_t)(q - vi.cellbase);
        const uint32_t it = fdiv(local, vi.m_ns), is = local - it * (uint32_t)vi.ns;
        if ((int)it >= vi.nt) continue;  // padding of the view's last chunk
        const unsigned long long ro = ((unsigned long long)vi.rkv_hi << 32) | vi.rkv_lo;
                const short4 rk = ldg(S.rkv + ro + (uint32_t)((vi.t0 + (int)it) * S.Ws + vi.s0 + (int)is));
        int a[3] = {rk.x, rk.y, rk.z};
        if (h <= 4) {  // the usual heights: the levels' loads issue together
            uint2 w[4];
#pragma unroll
            for (int L = 0; L < 4; ++L) {
                w[L] = make_uint2(0u, 0u);
                if (L >= S.lmin && L < h) {
                    const int2 vo = ctl.voff[vw][L];
                    w[L] = acc[vo.x + (int)it * vo.y + (int)is];
                }
            }
#pragma unroll
            for (int L = 0; L < 4; ++L) {
                a[0] += (int)(int16_t)(w[L].x & 0xFFFFu);
                a[1] += (int)w[L].x >> 16;
                a[2] += (int)(int16_t)(w[L].y & 0xFFFFu);
            }
        } else {
            for (int L = S.lmin; L < h; ++L) {
                const int2 vo = ctl.voff[vw][L];
                const uint2 w = acc[vo.x + (int)it * vo.y + (int)is];
                a[0] += (int)(int16_t)(w.x & 0xFFFFu);
                a[1] += (int)w.x >> 16;
                a[2] += (int)(int16_t)(w.y & 0xFFFFu);
            }
        }
        const uint32_t c8 = ycocg_to_rgb8(a);
        // the patch aliases the record list: all B3 readers passed the barrier above
        patch[q] = make_float4((float)(c8 & 0xFFu), (float)((c8 >> 8) & 0xFFu), (float)((c8 >> 16) & 0xFFu), 0.f);
    }
    __syncthreads();
    PHASE_MARK(8);
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

#ifndef HMLFC_EST_SLACK
#define HMLFC_EST_SLACK 120
#endif
constexpr int kEstSlackPct = HMLFC_EST_SLACK;  // the full-tile pass is tried when the estimate is below this share of the arena

// reset of the accumulators the next pass's SV phase writes with atomics (callers: after a barrier that every reader has passed)
__device__ __forceinline__ void reset_ctl(Ctl &ctl)
{
    const int tid = threadIdx.x;
    if (tid < 4) { ctl.lo[tid] = 0x7fffffff; ctl.hi[tid] = -1; }
    if (tid == 32) ctl.n_rec = 0;
}

// ---------------------------------------------------------------------------------------------------------------
// Pixel mapping of a pass of pw x ph pixels at (ox, oy).  full: the whole TW x TH tile, thread (tid % (TW / 4), tid / (TW / 4)) owns 4
// consecutive pixels.  Otherwise a sub-tile of at most NT pixels, one pixel per thread (pixel slot 0).  One code path serves both
// (slots 1..3 are simply empty in sub-tile passes): the kernel is instruction-cache sensitive, so the phases exist once.
template <int kTW>
__device__ __forceinline__ void thread_pixel(int ox, int oy, bool full, int lpw, int npx, int &x0, int &y, int &npix)
{
    constexpr int kTPR = kTW / kPPL;
    const int tid = threadIdx.x;
    if (full) { x0 = ox + (tid % kTPR) * kPPL; y = oy + tid / kTPR; npix = kPPL; }
    else { x0 = ox + (tid & ((1 << lpw) - 1)); y = oy + (tid >> lpw); npix = tid < npx ? 1 : 0; }
}

// ---------------------------------------------------------------- A: rays of the thread's pixels
template <int kTW>
__device__ __forceinline__ void setup_rays(const DevStream &S, const Camera &cam, int W, int H, int ox, int oy, bool full, int lpw, int npx,
                                           PixTaps (&pt)[kPPL])
{
    constexpr int kTPR = kTW / kPPL, kCPL = kTW / 32, kRPW = 32 / kTPR;  // threads per tile row, tile columns per lane, tile rows per warp
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    int x0, y, npix;
    thread_pixel<kTW>(ox, oy, full, lpw, npx, x0, y, npix);
    // screen coordinates once per column / row of the tile, shared by shuffles (sub-tiles: each lane its own)
    float pxl[kCPL];
#pragma unroll
    for (int j = 0; j < kCPL; ++j) pxl[j] = ray_screen(cam.tan_half_x, W, full ? ox + lane * kCPL + j : x0);
    const float pyl = ray_screen(cam.tan_half_y, H, full ? oy + warp * kRPW + (lane % kRPW) : y);
    const float py = __shfl_sync(FULL, pyl, full ? lane / kTPR : lane);
#pragma unroll
    for (int p = 0; p < kPPL; ++p) {
        // pixel column (tid % kTPR) * 4 + p of the tile was computed by lane column / kCPL as its value column % kCPL
        const float px = __shfl_sync(FULL, pxl[kCPL == 1 ? 0 : (p & (kCPL - 1))], full ? ((lane % kTPR) * kPPL + p) / kCPL : lane);
        pt[p] = pixel_taps(S, cam, px, py, p < npix && x0 + p < W && y < H);
    }
}


// ---------------------------------------------------------------------------------------------------------------
// One pass over a (sub-)tile whose rays are set up: ranges (SV), tables (T), decode (decode_patch), gather + blend (C).
// Returns true (CTA-uniform) when rgb[] holds the pass's pixels (background where the ray misses); false when the
// tables do not fit the arena and the (sub-)tile must be split.
template <int kArenaBytes, int kNT, bool kSubpel = false, bool kCs = false>
__device__ __forceinline__ bool tile_pass(const DevStream &S, Ctl &ctl, unsigned char *__restrict__ arena, const PixTaps (&pt)[kPPL],
                                          uint32_t (&rgb)[kPPL])
{
    constexpr int PPL = kPPL;
    constexpr int kSpecZero = kNT == 256 ? 1536 : (kNT == 512 ? 3072 : 6144);  // 16-byte words zeroed while warps 0 and 1 build the tables
    const int lane = threadIdx.x & 31;
    __syncthreads();  // the previous pass's readers of ctl / the patch are done; ctl's accumulators are reset (kernel start / end of the last pass)
    PHASE_MARK(1);

    // ------------------------------------------------------------ SV: (u,v) range and (s,t) box of the pass's taps
    int ls0 = 0x7fffffff, lt0 = 0x7fffffff, ls1 = -1, lt1 = -1;
    int ulo = 0x7fffffff, vlo = 0x7fffffff, uhi = -1, vhi = -1;
#pragma unroll
    for (int p = 0; p < PPL; ++p)
        if (pt[p].uv != kNone) {
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
    if (uhi >= 0) {
        if (lane < 4) atomicMin(&ctl.lo[lane], lane == 0 ? ulo : lane == 1 ? vlo : lane == 2 ? ws0 : wt0);
        else if (lane < 8) atomicMax(&ctl.hi[lane - 4], lane == 4 ? uhi : lane == 5 ? vhi : lane == 6 ? ws1 : wt1);
    }
    __syncthreads();
    PHASE_MARK(3);
    const int bu0 = ctl.lo[0], bv0 = ctl.lo[1], bs0 = ctl.lo[2], bt0 = ctl.lo[3];
    const int bs1 = ctl.hi[2], bt1 = ctl.hi[3];
    const int nu = ctl.hi[0] - bu0 + 1, nv = ctl.hi[1] - bv0 + 1;
    bool go = true, done = false;
    if (ctl.hi[0] < 0) { go = false; done = true; }  // no ray of the sub-tile hits the slab: background only
    else if (nu > kMaxV || nv > kMaxV) { PASS_STAT(8); go = false; }
    else {
        // Early exit before the tables are built: from the pass's exact (u,v) range and (s,t) box, cells ~ (2 ns + nu)
        // (2 nt + nv) (every pixel touches 2 x 2 views) and accumulator samples ~ cells (level 0) + box area x planes
        // of every level >= 1.  Only a hint (tables_fit decides): a pass that is let through and does not fit is
        // split after the tables are built, one that is split needlessly costs some halo.
        const int ns = bs1 - bs0 + 1, nt = bt1 - bt0 + 1;
        const int area = ns * nt;
        const int cells = (2 * ns + nu) * (2 * nt + nv) + 16 * nu * nv;
        int accs = cells;
        for (int L = 1; L < S.h; ++L)
            accs += area * ((((bu0 + nu - 1) >> L) - (bu0 >> L) + 1) * (((bv0 + nv - 1) >> L) - (bv0 >> L) + 1));
        if (16 * cells + 8 * accs > kArenaBytes / 100 * kEstSlackPct) { PASS_STAT(9); go = false; }
    }
    if (!go) {
        __syncthreads();  // every thread has read the ranges
        reset_ctl(ctl);
        return done;
    }

    // -------------------------------------------------------- T: tables (warp 0: views, warp 1: planes; the others zero the head of the
    // accumulator region, whose size is not known yet)
    {
        const int tid = threadIdx.x, warp = tid >> 5;
        TileHeader rg;
        rg.bu0 = bu0; rg.bv0 = bv0; rg.nu = nu; rg.nv = nv; rg.bs0 = bs0; rg.bs1 = bs1; rg.bt0 = bt0; rg.bt1 = bt1;
        if (warp == 0) build_view_table(S, ctl.aff, rg, ctl.tab);
        else if (warp == 1) build_slot_table(S, ctl.aff, rg, ctl.tab);
        else {
            uint4 *z = reinterpret_cast<uint4 *>(arena);
            for (int q = tid - 64; q < kSpecZero; q += kNT - 64) z[q] = make_uint4(0u, 0u, 0u, 0u);
        }
    }
    __syncthreads();
    PHASE_MARK(4);
    bool ok = tables_fit<kArenaBytes>(ctl.tab.hdr);
    if (!ok) PASS_STAT(10);
    else ok = decode_patch<kArenaBytes, kNT, kSubpel, kCs>(S, ctl, arena, kSpecZero);
    reset_ctl(ctl);  // behind a barrier that followed every read of the ranges and of the record count
    if (!ok) return false;

    // ------------------------------------------------ C: gather + blend
    const float4 *patch = reinterpret_cast<const float4 *>(arena + (((size_t)ctl.tab.hdr.nacc * 8 + 15) & ~(size_t)15));
#pragma unroll
    for (int p = 0; p < PPL; ++p)
        if (pt[p].uv != kNone) rgb[p] = blend_pixel(S, ctl, patch, pt[p], bu0, bv0);
    PHASE_MARK(9);
    return true;
}


// ---------------------------------------------------------------------------------------------------------------
// One tile by the general path: the whole tile (4 pixels per thread); if it does not fit (low magnification: more light-field samples
// than output pixels under the tile), its four quadrants with one pixel per thread, each split again when it does not fit; a sub-tile of
// the last level that still does not fit (strong minification) is rendered by 16 direct sample decodes per pixel.  ctl.cam, ctl.aff and
// ctl.lut are set and visible, the accumulators of ctl are reset (reset_ctl).  path = child index (2 bits) of every level on the way down.
template <int kArenaBytes, int kNT, int kTW, bool kSubpel = false, bool kCs = false>
__device__ __forceinline__ void render_tile_general(const DevStream &S, Ctl &ctl, unsigned char *__restrict__ arena, int W, int H, uint8_t *__restrict__ out,
                                                    int out_aligned, int view, int tile_x, int tile_y)
{
    constexpr int kTH = kNT * kPPL / kTW;
    constexpr int kLMax = kTW == 64 && kTH == 64 ? 3 : 2;  // quadtree levels below the tile: the smallest sub-tile is 8 pixels wide or high
    const Camera &cam = ctl.cam;
    const uint32_t bg = (uint32_t)S.bg[0] | ((uint32_t)S.bg[1] << 8) | ((uint32_t)S.bg[2] << 16);
    int lvl = 0;
    uint32_t path = 0u;
    for (;;) {
        int sx = tile_x * kTW, sy = tile_y * kTH;
        for (int l = 1; l <= lvl; ++l) {
            const uint32_t c = (path >> (2 * (l - 1))) & 3u;
            sx += (int)(c & 1u) * (kTW >> l); sy += (int)(c >> 1) * (kTH >> l);
        }
        const bool full = lvl == 0;
        const int lpw = 31 - __clz(kTW >> lvl), npx = (kTW >> lvl) * (kTH >> lvl);
        bool done = true;
        if (sx < W && sy < H) {
            PixTaps pt[kPPL];
            uint32_t rgb[kPPL];
#pragma unroll
            for (int p = 0; p < kPPL; ++p) rgb[p] = bg;
            PHASE_MARK(-1);
            setup_rays<kTW>(S, cam, W, H, sx, sy, full, lpw, npx, pt);
            PHASE_MARK(0);
            PASS_STAT(lvl);
            done = tile_pass<kArenaBytes, kNT, kSubpel, kCs>(S, ctl, arena, pt, rgb);
            if (done) PASS_STAT(4 + lvl);
            if (!done && lvl == kLMax) {
                PASS_STAT(13);
                if (pt[0].uv != kNone) rgb[0] = direct_pixel(S, pt[0]);
                done = true;
            }
            if (done) {
                int x0, y, npix;
                thread_pixel<kTW>(sx, sy, full, lpw, npx, x0, y, npix);
                if (full) store4(out, view, W, H, x0, y, rgb, out_aligned);
                else store1(out, view, W, H, x0, y, npix > 0, rgb[0], out_aligned);
                PHASE_MARK(10);
            }
        }
        if (!done) { ++lvl; path &= ~(3u << (2 * (lvl - 1))); continue; }  // descend to the first child
        while (lvl > 0 && ((path >> (2 * (lvl - 1))) & 3u) == 3u) --lvl;       // last child done: back to the parent's level
        if (lvl == 0) break;
        path += 1u << (2 * (lvl - 1));
    }
}

}  // namespace

}  // namespace hmlfc
